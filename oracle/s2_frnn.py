"""S2 fixed-radius nearest-neighbour graph in the latent space ("a
fixed-radius algorithm builds connections between spacepoints in this latent space
(edges)"; line 87 names the FRNN package).  BASELINE.json configs[0]: "radius set by the
oracle for mean degree D, cap K, ties to lower index, edges directed inner->outer r".

Definition used (readings C-7, C-8, C-9, C-11 of SURVEY.md section 8(c)):
  for every hit i, candidates are the hits j != i of the SAME event with outer(i, j) and
      d2(i,j) = sum_{k=0}^{d_e-1} (e_ik - e_jk)^2  <=  r^2
  evaluated in fp64 from the fp32 embedding, k ascending, separate multiply and add,
  r^2 = (double)r_fp32 squared in fp64;
  outer(i, j)  <=>  (r_i, |z_i|, i) < (r_j, |z_j|, j) lexicographically on the fp32 features;
  if more than K candidates, keep the K smallest by (d2, j);  emit the directed edge i -> j.
Output: src, dst int32 sorted by (src, dst), rowptr int32 [N+1].

Two implementations: `frnn_brute` (the definition, O(N^2) per event) and `frnn_grid`
(candidates from the 3^g neighbouring cells of a grid on the first g <= 3 latent
coordinates with cell edge >= r; every pair within r differs by at most one cell per axis,
so the result is identical).  tests/test_oracle_frnn.py cross-checks them on every event of
2k hits or fewer (BASELINE.json north_star) and pins the decision rule with closed forms
and a pure-Python triple loop.
"""
from __future__ import annotations

import numpy as np


def radius_squared(r_f32) -> float:
    r = float(np.float32(r_f32))
    return r * r


def dist2(eq, ec):
    """[Q,d] x [C,d] fp64 -> [Q,C]; k ascending, multiply then add (no fused operation in numpy)."""
    d2 = np.zeros((eq.shape[0], ec.shape[0]), dtype=np.float64)
    for k in range(eq.shape[1]):
        diff = eq[:, k, None] - ec[None, :, k]
        d2 = d2 + diff * diff
    return d2


def outer_mask(hits_f32, qi, cj):
    """outer(i,j) for all i in qi, j in cj (global indices)."""
    r = hits_f32[:, 0]
    az = np.abs(hits_f32[:, 2])
    ri, rj = r[qi][:, None], r[cj][None, :]
    zi, zj = az[qi][:, None], az[cj][None, :]
    ii, jj = np.asarray(qi)[:, None], np.asarray(cj)[None, :]
    return (ri < rj) | ((ri == rj) & ((zi < zj) | ((zi == zj) & (ii < jj))))


def _search_block(emb64, hits_f32, qi, cj, r2, K):
    """Neighbour lists of the queries qi among the candidates cj (ascending global indices).
    Returns list of (dst ascending, d2) per query."""
    d2 = dist2(emb64[qi], emb64[cj])
    ok = outer_mask(hits_f32, qi, cj) & (d2 <= r2)
    out = []
    for a in range(len(qi)):
        c = np.nonzero(ok[a])[0]                 # ascending candidate position == ascending j
        if len(c) > K:
            order = np.argsort(d2[a, c], kind="stable")[:K]   # ties in d2 -> lower j first
            c = np.sort(c[order])
        out.append((cj[c], d2[a, c]))
    return out


def _assemble(n, per_query, return_d2):
    deg = np.array([len(p[0]) for p in per_query], dtype=np.int64)
    rowptr = np.zeros(n + 1, dtype=np.int64)
    rowptr[1:] = np.cumsum(deg)
    src = np.repeat(np.arange(n, dtype=np.int64), deg).astype(np.int32)
    dst = (np.concatenate([p[0] for p in per_query]) if n else np.zeros(0)).astype(np.int32)
    if return_d2:
        d2 = np.concatenate([p[1] for p in per_query]) if n else np.zeros(0)
        return src, dst, rowptr.astype(np.int32), d2
    return src, dst, rowptr.astype(np.int32)


def frnn_brute(emb_f32, hits_f32, event_offsets, r_f32, K, chunk=256, return_d2=False):
    emb64 = np.asarray(emb_f32, np.float32).astype(np.float64)
    hits_f32 = np.asarray(hits_f32, np.float32)
    n = emb64.shape[0]
    r2 = radius_squared(r_f32)
    per_query = [None] * n
    for b in range(len(event_offsets) - 1):
        lo, hi = int(event_offsets[b]), int(event_offsets[b + 1])
        cj = np.arange(lo, hi)
        for q0 in range(lo, hi, chunk):
            qi = np.arange(q0, min(q0 + chunk, hi))
            for i, res in zip(qi, _search_block(emb64, hits_f32, qi, cj, r2, K)):
                per_query[i] = res
    return _assemble(n, per_query, return_d2)


def frnn_grid(emb_f32, hits_f32, event_offsets, r_f32, K, g=3, return_d2=False, max_block=1 << 22):
    emb64 = np.asarray(emb_f32, np.float32).astype(np.float64)
    hits_f32 = np.asarray(hits_f32, np.float32)
    n, d_e = emb64.shape
    g = min(g, d_e)
    r2 = radius_squared(r_f32)
    cell = float(np.float32(r_f32)) * (1.0 + 1e-9)
    per_query = [None] * n
    for b in range(len(event_offsets) - 1):
        lo, hi = int(event_offsets[b]), int(event_offsets[b + 1])
        if hi == lo:
            continue
        if cell <= 0.0:
            for i in range(lo, hi):
                per_query[i] = (np.zeros(0, np.int64), np.zeros(0))
            continue
        x = emb64[lo:hi, :g]
        c = np.floor((x - x.min(axis=0)) / cell).astype(np.int64)          # [Nb, g] cell coordinates
        dims = c.max(axis=0) + 1
        if float(np.prod(dims.astype(np.float64))) > 2.0 ** 62:
            raise ValueError("grid too fine for this radius")
        strides = np.concatenate([[1], np.cumprod(dims[:-1])])
        cid = c @ strides
        order = np.argsort(cid, kind="stable")                              # ascending hit index inside a cell
        ucid, start = np.unique(cid[order], return_index=True)
        end = np.append(start[1:], len(order))
        members = {int(u): order[s:e] + lo for u, s, e in zip(ucid, start, end)}
        coords = {int(u): c[order[s]] for u, s in zip(ucid, start)}
        offsets = np.stack(np.meshgrid(*[[-1, 0, 1]] * g, indexing="ij"), axis=-1).reshape(-1, g)
        for u, qi in members.items():
            cc = coords[u]
            neigh = []
            for o in offsets:
                nc = cc + o
                if np.any(nc < 0) or np.any(nc >= dims):
                    continue
                m = members.get(int(nc @ strides))
                if m is not None:
                    neigh.append(m)
            cj = np.sort(np.concatenate(neigh))
            step = max(1, max_block // max(1, len(cj)))
            for q0 in range(0, len(qi), step):
                qq = qi[q0:q0 + step]
                for i, res in zip(qq, _search_block(emb64, hits_f32, qq, cj, r2, K)):
                    per_query[i] = res
    return _assemble(n, per_query, return_d2)


def frnn(emb_f32, hits_f32, event_offsets, r_f32, K, return_d2=False):
    """Brute force up to 2k hits per event, grid search above (BASELINE.json north_star)."""
    sizes = np.diff(np.asarray(event_offsets))
    f = frnn_brute if (len(sizes) == 0 or sizes.max() <= 2000) else frnn_grid
    return f(emb_f32, hits_f32, event_offsets, r_f32, K, return_d2=return_d2)
