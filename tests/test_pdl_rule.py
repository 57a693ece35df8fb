"""-m "not gpu": every kernel launched through TRK_LAUNCH starts with TRK_GRID_DEP_WAIT().

TRK_LAUNCH (csrc/common.cuh) sets programmatic stream serialization on every launch, so a kernel may start while its
predecessor in the stream is still draining; it is correct only if griddepcontrol.wait is executed by all threads before
any memory access or early return.  A kernel added without it would race only under load and pass the small tests, so the
rule is enforced on the source text: the first statement of every __global__ body is the wait.  csrc/cc_noalloc.cu launches
with <<< >>> (no such attribute) and is exempt.
"""
import os
import re

CSRC = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2501_05520_b200", "csrc")
EXEMPT = {"cc_noalloc.cu"}


def _strip_comments(text):
    text = re.sub(r"/\*.*?\*/", lambda m: " " * len(m.group(0)), text, flags=re.S)
    return re.sub(r"//[^\n]*", lambda m: " " * len(m.group(0)), text)


def _match_paren(text, i):
    depth = 0
    while True:
        depth += {"(": 1, ")": -1}.get(text[i], 0)
        i += 1
        if depth == 0:
            return i


def _kernels(text):
    """(name, body start) of every __global__ function definition."""
    for m in re.finditer(r"__global__", text):
        i = text.index("(", m.end())
        while re.search(r"__(launch_bounds|cluster_dims)__\s*$", text[m.end():i]):   # attribute(..) before the name: skip it
            i = text.index("(", _match_paren(text, i))
        name = re.findall(r"([A-Za-z_][A-Za-z0-9_]*)\s*$", text[:i])[0]
        j = _match_paren(text, i)
        rest = text[j:]
        k = len(rest) - len(rest.lstrip())
        if rest[k] == ";":                                  # a declaration
            continue
        assert rest[k] == "{", (name, rest[k:k + 40])
        yield name, j + k + 1


def test_every_trk_launch_kernel_waits_first():
    found = 0
    for f in sorted(os.listdir(CSRC)):
        if not f.endswith((".cu", ".cuh")) or f in EXEMPT:
            continue
        text = _strip_comments(open(os.path.join(CSRC, f)).read())
        for name, start in _kernels(text):
            found += 1
            assert text[start:].lstrip().startswith("TRK_GRID_DEP_WAIT();"), f"{f}: kernel {name} does not start with TRK_GRID_DEP_WAIT()"
    assert found >= 45, found          # 48 kernel definitions (templates once) at the time of writing
