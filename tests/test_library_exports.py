"""-m "not gpu": libtrk.so builds, loads and exports every symbol include/trk.h declares (no compute calls)."""
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_build_and_exports():
    import __graft_entry__
    __graft_entry__.build()
    from paper_2501_05520_b200 import EXPORTS, lib
    L = lib()
    header = open(os.path.join(ROOT, "include", "trk.h")).read()
    declared = set(re.findall(r"\b(trk_[a-z0-9_]+)\s*\(", header))
    assert declared == set(EXPORTS), declared ^ set(EXPORTS)
    for name in declared:
        assert hasattr(L, name), name
    assert L.trk_status_string(0) == b"TRK_OK" and L.trk_status_string(6) == b"TRK_ERR_UNSUPPORTED_DEVICE"


def test_config_struct_matches_header_size():
    """The ctypes mirror of trk_config must have the C layout (checked against a compiled sizeof)."""
    import ctypes
    import subprocess
    import tempfile
    from paper_2501_05520_b200.binding import TrkBatch, TrkConfig, TrkMlp, TrkResult
    src = '#include <stdio.h>\n#include "trk.h"\nint main(){printf("%zu %zu %zu %zu\\n",sizeof(trk_mlp),sizeof(trk_config),sizeof(trk_batch),sizeof(trk_result));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "s")
        subprocess.check_call(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), c, "-o", exe])
        sizes = [int(v) for v in subprocess.check_output([exe]).split()]
    assert sizes == [ctypes.sizeof(TrkMlp), ctypes.sizeof(TrkConfig), ctypes.sizeof(TrkBatch), ctypes.sizeof(TrkResult)]


def test_create_fails_loudly_without_a_gpu_or_with_bad_config():
    import numpy as np
    import torch
    from paper_2501_05520_b200 import TrkError, trk_from_config
    from synth.configs import get_config, load_calibration
    from synth.weights import make_model
    cfg = get_config("toy")
    model = make_model(cfg)
    calib = load_calibration("toy")
    try:
        t = trk_from_config(cfg, model, calib, max_hits=100)
        assert torch.cuda.is_available(), "trk_create must not succeed without a device"
        t.close()
    except TrkError as e:
        assert not torch.cuda.is_available() and e.status in (4, 6)
    bad = dict(model, filter=dict(model["filter"], dims=[7, 64, 1], weight=[np.zeros((64, 7), np.float32), model["filter"]["weight"][1]]))
    try:
        trk_from_config(cfg, bad, calib, max_hits=100)
        assert False, "shape error expected"
    except TrkError as e:
        assert e.status in (2, 4, 6)


def test_cc_noalloc_refuses_bad_sizes_on_the_host():
    """trk_cc_noalloc checks its arguments before it touches the CUDA runtime: a size beyond its built-in scratch array is
    TRK_ERR_CAPACITY with a message that names the limit, bad arguments are TRK_ERR_INVALID_ARG, n == 0 is a no-op --
    all without a device (the binding's constant must equal the header's)."""
    import ctypes
    from paper_2501_05520_b200 import CC_NOALLOC_MAX_HITS, lib
    header = open(os.path.join(ROOT, "include", "trk.h")).read()
    assert int(re.search(r"#define\s+TRK_CC_NOALLOC_MAX_HITS\s+(\d+)", header).group(1)) == CC_NOALLOC_MAX_HITS
    L = lib()
    null = ctypes.c_void_p(0)
    junk = ctypes.c_void_p(256)                      # never dereferenced: every call below is refused or empty
    assert L.trk_cc_noalloc(CC_NOALLOC_MAX_HITS + 1, junk, junk, junk, 1, 0.5, junk, null) == 3
    assert b"TRK_CC_NOALLOC_MAX_HITS" in L.trk_last_error(None)
    assert L.trk_cc_noalloc(-1, junk, junk, junk, 0, 0.5, junk, null) == 1
    assert L.trk_cc_noalloc(10, null, junk, junk, 5, 0.5, junk, null) == 1
    assert L.trk_cc_noalloc(10, junk, junk, junk, 5, 0.5, null, null) == 1
    assert L.trk_cc_noalloc(0, null, null, null, 0, 0.5, null, null) == 0
