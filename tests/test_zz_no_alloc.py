"""-m gpu: trk_cc_noalloc, the S5 entry point for callers that cannot allocate device memory.

Such callers exist around a served tracking backend: the serving framework owns the GPU and gives the backend a fixed
memory budget, some code runs where cudaMalloc is forbidden or stalls the whole device (a stream
capture open elsewhere in the process, a stream host callback), and tight loops cannot pay cudaMalloc's implicit
synchronisation.  trk_create allocates, so they cannot hold a context; trk_cc_noalloc keeps its union-find scratch in a
fixed array inside libtrk.so instead (limit: TRK_CC_NOALLOC_MAX_HITS hits).

What is checked: its labels equal those of the existing context path (trk_stage_cc) bit for bit -- the bar every S5 test
of this repository uses, labels being integers -- on two calls in a row, the second on a smaller, different graph, so that
whatever the first call left in the shared scratch would show; and a size beyond the limit is refused before any launch.

The file name sorts last on purpose: pytest -x stops at the first failure, so a failure here hides no other test.  It
needs nothing from the tests before it (own inputs, own context) and passes alone in a fresh process as well.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _track_like_graph(n, n_edges, seed):
    """Random chains plus random cross links with uniform scores: many components of mixed size, some of them merged by
    high-score cross links -- the shape of an S4 output.  Pure input generation, none of the method's arithmetic."""
    rng = np.random.default_rng(seed)
    perm = rng.permutation(n).astype(np.int32)
    chain_src, chain_dst = perm[:-1], perm[1:]
    breaks = rng.random(n - 1) < 0.12                                  # chains of ~8 hits
    chain_src, chain_dst = chain_src[~breaks], chain_dst[~breaks]
    extra = max(n_edges - len(chain_src), 0)
    src = np.concatenate([chain_src, rng.integers(0, n, extra, dtype=np.int32)])
    dst = np.concatenate([chain_dst, rng.integers(0, n, extra, dtype=np.int32)])
    score = rng.random(len(src)).astype(np.float32)
    score[: len(chain_src)] = 0.5 + 0.5 * score[: len(chain_src)]        # chain edges mostly pass the cut
    score[len(chain_src):] *= 0.52                                       # a few cross links pass too
    order = np.lexsort((dst, src))
    return src[order], dst[order], score[order]


def _context(max_hits):
    from paper_2501_05520_b200 import trk_from_config
    from synth.configs import get_config, load_calibration
    from synth.weights import make_model
    cfg = get_config("toy")
    return trk_from_config(cfg, make_model(cfg), load_calibration("toy"), max_hits=max_hits)


def test_cc_noalloc_matches_context_path_on_two_calls_in_a_row():
    import torch
    from oracle import s5_cc
    from paper_2501_05520_b200 import cc_noalloc
    cut = 0.5
    trk = _context(60000)
    try:
        for n, n_edges, seed in ((60000, 90000, 11), (20011, 26000, 12)):     # second call: smaller, other graph
            src, dst, score = _track_like_graph(n, n_edges, seed)
            d = [torch.from_numpy(a).cuda() for a in (src, dst, score)]
            want = trk.stage_cc(n, d[0], d[1], d[2], cut)
            got = torch.full((n,), -7, dtype=torch.int32, device="cuda")       # caller-owned output, pre-filled with junk
            cc_noalloc(n, d[0], d[1], d[2], cut, got)
            torch.cuda.synchronize()
            assert torch.equal(got, want), f"n={n}: {(got != want).sum().item()} labels differ from trk_stage_cc"
            ref = s5_cc.connected_components(n, src, dst, score, cut)
            assert np.array_equal(got.cpu().numpy(), ref)
            assert 1000 < len(np.unique(ref)) < n                              # neither trivial nor one blob
    finally:
        trk.close()


def test_cc_noalloc_refuses_sizes_beyond_its_scratch_and_accepts_the_limit():
    import torch
    from paper_2501_05520_b200 import CC_NOALLOC_MAX_HITS, TrkError, cc_noalloc
    n = CC_NOALLOC_MAX_HITS
    labels = torch.full((n + 1,), -7, dtype=torch.int32, device="cuda")
    e = torch.zeros(1, dtype=torch.int32, device="cuda")
    s = torch.ones(1, dtype=torch.float32, device="cuda")
    with pytest.raises(TrkError) as err:
        cc_noalloc(n + 1, e, e, s, 0.5, labels)
    assert err.value.status == 3 and "TRK_CC_NOALLOC_MAX_HITS" in str(err.value)      # TRK_ERR_CAPACITY, says why
    torch.cuda.synchronize()
    assert bool((labels == -7).all()), "a refused call must not enqueue anything"
    # exactly the limit: a chain over the last hits, so the top of the scratch array is used
    src = torch.arange(n - 1000, n - 1, dtype=torch.int32, device="cuda")
    dst = src + 1
    sc = torch.ones(src.numel(), dtype=torch.float32, device="cuda")
    cc_noalloc(n, src, dst, sc, 0.5, labels)
    torch.cuda.synchronize()
    want = torch.arange(n, dtype=torch.int32, device="cuda")
    want[n - 1000:] = n - 1000
    assert torch.equal(labels[:n], want) and int(labels[n]) == -7
