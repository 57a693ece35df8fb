"""S5 weakly-connected components ("the GNN edge scores are passed to the
weekly-connected-component (WCC) algorithm to form track candidates"; line 87: Boost graph).
Kept = {k : score_k > cut} (strict, reading C-11); direction ignored;
label[v] = smallest global hit index in v's component (reading C-17), singletons label themselves.

Two implementations: union-find (used) and BFS in index order (the cross-check BASELINE.json asks for).
Pure-Python loops: O(E) dictionary-free array walks, a few seconds per million edges.
"""
from __future__ import annotations

from collections import deque

import numpy as np


def labels_union_find(n, src, dst, keep=None):
    src = np.asarray(src, np.int64)
    dst = np.asarray(dst, np.int64)
    if keep is not None:
        keep = np.asarray(keep, bool)
        src, dst = src[keep], dst[keep]
    parent = list(range(n))
    for a, b in zip(src.tolist(), dst.tolist()):
        while parent[a] != a:
            parent[a] = parent[parent[a]]
            a = parent[a]
        while parent[b] != b:
            parent[b] = parent[parent[b]]
            b = parent[b]
        if a != b:
            if a < b:                 # the smaller index becomes the root, so root == min of the set
                parent[b] = a
            else:
                parent[a] = b
    out = np.empty(n, dtype=np.int32)
    for v in range(n):
        r = v
        while parent[r] != r:
            r = parent[r]
        out[v] = r
    return out


def labels_bfs(n, src, dst, keep=None):
    src = np.asarray(src, np.int64)
    dst = np.asarray(dst, np.int64)
    if keep is not None:
        keep = np.asarray(keep, bool)
        src, dst = src[keep], dst[keep]
    adj = [[] for _ in range(n)]
    for a, b in zip(src.tolist(), dst.tolist()):
        adj[a].append(b)
        adj[b].append(a)
    label = [-1] * n
    for v in range(n):                # index order, so the first vertex reached is the component minimum
        if label[v] >= 0:
            continue
        label[v] = v
        q = deque([v])
        while q:
            u = q.popleft()
            for w in adj[u]:
                if label[w] < 0:
                    label[w] = v
                    q.append(w)
    return np.asarray(label, dtype=np.int32)


def connected_components(n, src, dst, scores, cut_f32):
    keep = np.asarray(scores).astype(np.float32) > np.float32(cut_f32)   # fp32 interchange values
    return labels_union_find(n, src, dst, keep)
