"""Pins for the oracle's S5 (SURVEY.md section 8(c) "Pins / S5 CC")."""
import numpy as np
import scipy.sparse as sp
from scipy.sparse.csgraph import connected_components as scipy_cc

from oracle import s5_cc
from synth.events import generate_event, truth_edges


def test_closed_forms():
    uf = s5_cc.labels_union_find
    assert list(uf(5, [], [])) == [0, 1, 2, 3, 4]                                   # empty graph
    assert list(uf(5, [3, 2, 1, 0], [4, 3, 2, 1])) == [0] * 5                       # path
    assert list(uf(6, [5, 5, 5], [1, 2, 3])) == [0, 1, 1, 1, 4, 1]                  # star centred at 5 -> min is 1
    a = [(i, j) for i in range(3) for j in range(3) if i < j]
    b = [(i, j) for i in range(3, 7) for j in range(3, 7) if i < j]
    s, d = zip(*(a + b))
    assert list(uf(8, s, d)) == [0, 0, 0, 3, 3, 3, 3, 7]                            # two cliques + singleton
    assert list(uf(4, [0, 1], [1, 0])) == [0, 0, 2, 3]                              # both directions, weakly connected
    assert list(uf(3, [1], [1])) == [0, 1, 2]                                       # self loop
    assert list(uf(0, [], [])) == []


def test_union_find_equals_bfs_and_library():
    """BASELINE.json north_star: connected components against BFS; scipy as a library cross-check."""
    rng = np.random.default_rng(0)
    for n, e in [(1, 0), (50, 20), (300, 200), (300, 2000), (2000, 1500)]:
        src = rng.integers(0, n, e); dst = rng.integers(0, n, e)
        keep = rng.uniform(size=e) < 0.7
        a = s5_cc.labels_union_find(n, src, dst, keep)
        b = s5_cc.labels_bfs(n, src, dst, keep)
        assert np.array_equal(a, b) and a.dtype == np.int32
        assert np.all(a <= np.arange(n)) and np.array_equal(a[a], a)
        assert np.all(a[src[keep]] == a[dst[keep]])
        g = sp.coo_matrix((np.ones(keep.sum()), (src[keep], dst[keep])), shape=(n, n))
        ncomp, lab = scipy_cc(g, directed=True, connection="weak")
        assert ncomp == len(np.unique(a))
        mins = np.full(ncomp, n); np.minimum.at(mins, lab, np.arange(n))
        assert np.array_equal(a, mins[lab])


def test_invariances():
    rng = np.random.default_rng(1)
    n, e = 400, 500
    src = rng.integers(0, n, e); dst = rng.integers(0, n, e)
    a = s5_cc.labels_union_find(n, src, dst)
    p = rng.permutation(e)
    assert np.array_equal(a, s5_cc.labels_union_find(n, src[p], dst[p]))                 # edge order
    assert np.array_equal(a, s5_cc.labels_union_find(n, dst, src))                       # direction
    same = np.nonzero(a == a[src[0]])[0]
    assert np.array_equal(a, s5_cc.labels_union_find(n, np.append(src, same[0]), np.append(dst, same[-1])))  # intra-component edge


def test_cut_is_strict_fp32():
    lab = s5_cc.connected_components(4, [0, 1, 2], [1, 2, 3], np.array([0.5, 0.50000006, 0.49]), 0.5)
    assert list(lab) == [0, 1, 1, 3]


def test_truth_graph_partition_equals_particle_ids():
    e = generate_event(300, 0.1, 2)
    s, d = truth_edges(e["particle_id"], e["layer"], e["hits"])
    lab = s5_cc.labels_union_find(len(e["hits"]), s, d)
    pid = e["particle_id"]
    for p in np.unique(pid[pid >= 0]):
        idx = np.nonzero(pid == p)[0]
        assert np.all(lab[idx] == idx.min())
    noise = np.nonzero(pid < 0)[0]
    assert np.array_equal(lab[noise], noise)
