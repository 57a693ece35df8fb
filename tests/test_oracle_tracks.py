"""Pins for the oracle's S6 track-candidate lists."""
import numpy as np

from oracle import s5_cc, s6_tracks
from synth.events import generate_event, truth_edges


def test_closed_forms():
    bt = s6_tracks.build_tracks
    off, hit = bt([0, 0, 2, 0, 2, 5], 2)                       # {0,1,3} {2,4} {5}
    assert off.tolist() == [0, 3, 5] and hit.tolist() == [0, 1, 3, 2, 4]
    off, hit = bt([0, 0, 2, 0, 2, 5], 3)
    assert off.tolist() == [0, 3] and hit.tolist() == [0, 1, 3]
    off, hit = bt([0, 0, 2, 0, 2, 5], 1)                       # every component is a track, singletons too
    assert off.tolist() == [0, 3, 5, 6] and hit.tolist() == [0, 1, 3, 2, 4, 5]
    off, hit = bt([0, 0, 2, 0, 2, 5], 4)
    assert off.tolist() == [0] and hit.tolist() == []
    off, hit = bt([], 1)
    assert off.tolist() == [0] and hit.tolist() == [] and off.dtype == np.int32 and hit.dtype == np.int32
    off, hit = bt([0, 1, 2], 0)                                # min_hits < 1 behaves like 1
    assert off.tolist() == [0, 1, 2, 3]


def test_against_lexsort_and_invariants():
    """A library sort as the cross-check: lexsort by (label, index), components filtered by bincount."""
    rng = np.random.default_rng(1)
    for n, e in [(1, 0), (40, 15), (500, 300), (3000, 2500)]:
        src = rng.integers(0, n, e); dst = rng.integers(0, n, e)
        lab = s5_cc.labels_union_find(n, src, dst)
        size = np.bincount(lab, minlength=n)
        for m in (1, 2, 3, 7):
            off, hit = s6_tracks.build_tracks(lab, m)
            order = np.lexsort((np.arange(n), lab))
            order = order[size[lab[order]] >= m]
            assert np.array_equal(hit, order.astype(np.int32))
            roots = np.flatnonzero((lab == np.arange(n)) & (size >= m))
            assert len(off) == len(roots) + 1 and off[0] == 0 and off[-1] == len(hit)
            assert np.array_equal(np.diff(off), size[roots])                  # track t is the t-th kept root, by label
            assert np.array_equal(hit[off[:-1]], roots.astype(np.int32))      # first hit of a track is its label
            assert len(np.unique(hit)) == len(hit)                            # a hit is in at most one track
            for t in range(len(roots)):
                seg = hit[off[t]:off[t + 1]]
                assert np.all(np.diff(seg) > 0) and np.all(lab[seg] == roots[t])


def test_truth_graph_gives_particles():
    """On the truth graph (consecutive same-particle hits) the tracks are exactly the particles' hit lists."""
    ev = generate_event(n_particles=200, noise_frac=0.1, seed=3)
    n = len(ev["hits"])
    src, dst = truth_edges(ev["particle_id"], ev["layer"], ev["hits"])
    lab = s5_cc.labels_union_find(n, src, dst)
    off, hit = s6_tracks.build_tracks(lab, 3)
    pid = ev["particle_id"]
    want = []
    for p in np.unique(pid[pid >= 0]):
        members = np.flatnonzero(pid == p)
        if len(members) >= 3:
            want.append(members)
    want.sort(key=lambda m: m[0])
    assert len(want) == len(off) - 1
    for t, m in enumerate(want):
        assert np.array_equal(hit[off[t]:off[t + 1]], m.astype(np.int32))
    assert not np.any(pid[hit] < 0)                                            # noise hits are in no track
