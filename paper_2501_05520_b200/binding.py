"""ctypes binding of include/trk.h: argument marshalling only -- every step of the path runs in
the CUDA kernels of libtrk.so.  torch is used for device memory and streams, nothing else.

There is no CPU fallback: if libtrk.so is missing or does not load, importing `lib()` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtrk.so")

TRK_FP32, TRK_BF16 = 0, 1
TRK_FILTER_RAW, TRK_FILTER_EMB = 0, 1

EXPORTS = [
    "trk_create", "trk_infer", "trk_destroy", "trk_infer_host", "trk_status_string", "trk_last_error",
    "trk_workspace_bytes", "trk_last_launch_count", "trk_stage_embed", "trk_stage_frnn", "trk_stage_filter",
    "trk_stage_compact", "trk_stage_gnn", "trk_stage_cc", "trk_gemm_bf16", "trk_profile_enable", "trk_profile_stage_ms", "trk_profile_kernel_ms",
    "trk_set_option", "trk_stage_tracks", "trk_infer_host_tracks", "trk_cc_noalloc", "trk_stage_gnn_csr",
]
CC_NOALLOC_MAX_HITS = 1048576  # TRK_CC_NOALLOC_MAX_HITS of include/trk.h

_f32p = C.POINTER(C.c_float)
_i32p = C.POINTER(C.c_int32)


class TrkMlp(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("dims", _i32p), ("weight", C.POINTER(_f32p)), ("bias", C.POINTER(_f32p))]


class TrkConfig(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("device", C.c_int32), ("precision", C.c_int32),
        ("embed", TrkMlp),
        ("frnn_radius", C.c_float), ("frnn_k", C.c_int32), ("grid_proj", _f32p), ("grid_dims", C.c_int32),
        ("filter", TrkMlp), ("filter_input", C.c_int32), ("filter_cut", C.c_float),
        ("gnn_hidden", C.c_int32), ("gnn_iters", C.c_int32), ("gnn_layernorm", C.c_int32),
        ("node_enc", TrkMlp), ("edge_enc", TrkMlp), ("edge_net", TrkMlp), ("node_net", TrkMlp), ("edge_dec", TrkMlp),
        ("gnn_cut", C.c_float),
        ("max_hits", C.c_int64), ("max_events", C.c_int64), ("max_cand_edges", C.c_int64), ("max_kept_edges", C.c_int64),
        ("min_track_hits", C.c_int32),
        ("filter_chunk_rows", C.c_int64), ("grid_max", C.c_int32),
    ]


class TrkBatch(C.Structure):
    _fields_ = [("n_events", C.c_int32), ("event_offsets", _i32p), ("hits", C.c_void_p)]


class TrkResult(C.Structure):
    _fields_ = [
        ("labels", C.c_void_p), ("counts", C.c_void_p),
        ("edge_src", C.c_void_p), ("edge_dst", C.c_void_p), ("edge_score", C.c_void_p), ("edge_capacity", C.c_int64),
        ("cand_src", C.c_void_p), ("cand_dst", C.c_void_p), ("cand_score", C.c_void_p), ("cand_capacity", C.c_int64),
        ("embedding", C.c_void_p),
        ("track_offsets", C.c_void_p), ("track_hits", C.c_void_p), ("track_counts", C.c_void_p), ("track_capacity", C.c_int64),
    ]


_lib = None


def lib():
    """Loads libtrk.so (raises if it is not built: the product has no other path)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2501_05520_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int32
    L.trk_create.argtypes = [C.POINTER(TrkConfig), C.POINTER(vp)]
    L.trk_infer.argtypes = [vp, C.POINTER(TrkBatch), C.POINTER(TrkResult), vp]
    L.trk_destroy.argtypes = [vp]
    L.trk_infer_host.argtypes = [vp, i32, _i32p, vp, vp, vp]
    L.trk_status_string.argtypes = [C.c_int]
    L.trk_status_string.restype = C.c_char_p
    L.trk_last_error.argtypes = [vp]
    L.trk_last_error.restype = C.c_char_p
    L.trk_workspace_bytes.argtypes = [vp]
    L.trk_workspace_bytes.restype = i64
    L.trk_last_launch_count.argtypes = [vp]
    L.trk_last_launch_count.restype = i64
    L.trk_stage_embed.argtypes = [vp, vp, i64, vp, vp]
    L.trk_stage_frnn.argtypes = [vp, vp, vp, _i32p, i32, vp, vp, vp, i64, vp, vp]
    L.trk_stage_filter.argtypes = [vp, vp, i64, vp, vp, i64, vp, vp]
    L.trk_stage_compact.argtypes = [vp, vp, vp, vp, i64, vp, vp, i64, vp, vp]
    L.trk_stage_gnn.argtypes = [vp, vp, i64, vp, vp, i64, vp, vp]
    L.trk_stage_cc.argtypes = [vp, i64, vp, vp, vp, i64, C.c_float, vp, vp]
    L.trk_gemm_bf16.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, i32, vp]
    L.trk_profile_enable.argtypes = [vp, i32]
    L.trk_set_option.argtypes = [vp, C.c_char_p, i64]
    L.trk_profile_stage_ms.argtypes = [vp, _f32p]
    L.trk_profile_kernel_ms.argtypes = [vp, _f32p, i32, _i32p, C.POINTER(i64)]
    L.trk_stage_tracks.argtypes = [vp, vp, i64, i32, vp, i64, vp, vp, vp]
    L.trk_infer_host_tracks.argtypes = [vp, i32, _i32p, vp, vp, vp, vp, vp]
    L.trk_stage_gnn_csr.argtypes = [vp, vp, i64, vp, vp, i64, vp, vp, vp, vp]
    L.trk_cc_noalloc.argtypes = [i64, vp, vp, vp, i64, C.c_float, vp, vp]
    for name in EXPORTS:
        if getattr(L, name).restype is C.c_int:
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


class TrkError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"{lib().trk_status_string(status).decode()}: {message}")
        self.status = status


def _mlp_struct(mlp, keep):
    dims = np.ascontiguousarray(mlp["dims"], dtype=np.int32)
    ws = [np.ascontiguousarray(w, dtype=np.float32) for w in mlp["weight"]]
    bs = [np.ascontiguousarray(b, dtype=np.float32) for b in mlp["bias"]]
    n = len(ws)
    wp = (_f32p * n)(*[w.ctypes.data_as(_f32p) for w in ws])
    bp = (_f32p * n)(*[b.ctypes.data_as(_f32p) for b in bs])
    keep += [dims, ws, bs, wp, bp]
    return TrkMlp(n, dims.ctypes.data_as(_i32p), wp, bp)


def _ptr(t):
    return C.c_void_p(0 if t is None else t.data_ptr())


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


class Trk:
    """One model instance: create once, infer many times, close."""

    def __init__(self, *, model, precision, frnn_radius, frnn_k, filter_input, filter_cut, gnn_hidden, gnn_iters, gnn_cut,
                 max_hits, max_events=1, max_cand_edges=None, max_kept_edges=None, gnn_layernorm=True, grid_proj=None,
                 grid_dims=None, device=0, min_track_hits=3, filter_chunk_rows=0, grid_max=0):
        L = lib()
        keep = []
        cfg = TrkConfig()
        cfg.struct_size = C.sizeof(TrkConfig)
        cfg.device = device
        cfg.precision = {"fp32": TRK_FP32, "bf16": TRK_BF16}.get(precision, precision)
        cfg.embed = _mlp_struct(model["embed"], keep)
        cfg.frnn_radius = float(frnn_radius)
        cfg.frnn_k = int(frnn_k)
        d_e = int(model["embed"]["dims"][-1])
        if grid_proj is not None:
            gp = np.ascontiguousarray(grid_proj, dtype=np.float32)
            keep.append(gp)
            cfg.grid_proj = gp.ctypes.data_as(_f32p)
            cfg.grid_dims = gp.shape[1]
        else:
            cfg.grid_proj = None
            cfg.grid_dims = min(3, d_e) if grid_dims is None else grid_dims
        cfg.filter = _mlp_struct(model["filter"], keep)
        cfg.filter_input = {"raw": TRK_FILTER_RAW, "emb": TRK_FILTER_EMB}.get(filter_input, filter_input)
        cfg.filter_cut = float(filter_cut)
        cfg.gnn_hidden, cfg.gnn_iters, cfg.gnn_layernorm = int(gnn_hidden), int(gnn_iters), int(bool(gnn_layernorm))
        for k in ("node_enc", "edge_enc", "edge_net", "node_net", "edge_dec"):
            setattr(cfg, k, _mlp_struct(model[k], keep))
        cfg.gnn_cut = float(gnn_cut)
        cfg.max_hits = int(max_hits)
        cfg.max_events = int(max_events)
        cfg.max_cand_edges = int(max_cand_edges if max_cand_edges is not None else max_hits * frnn_k)
        cfg.max_kept_edges = int(max_kept_edges if max_kept_edges is not None else cfg.max_cand_edges)
        cfg.min_track_hits = int(min_track_hits)
        cfg.filter_chunk_rows = int(filter_chunk_rows)
        cfg.grid_max = int(grid_max)
        self.cfg = cfg
        self.d_e = d_e
        self.device = device
        self._h = C.c_void_p()
        st = L.trk_create(C.byref(cfg), C.byref(self._h))
        if st != 0:
            raise TrkError(st, L.trk_last_error(None).decode())

    # ---- plumbing
    def _check(self, st):
        if st != 0:
            raise TrkError(st, lib().trk_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib().trk_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def workspace_bytes(self):
        return lib().trk_workspace_bytes(self._h)

    @property
    def last_launch_count(self):
        return lib().trk_last_launch_count(self._h)

    def set_option(self, key: str, value: int) -> None:
        """Per-context test / tuning hook (include/trk.h trk_set_option): kernel variants that compute the same result."""
        self._check(lib().trk_set_option(self._h, key.encode(), int(value)))

    def profile(self, on=True):
        self._check(lib().trk_profile_enable(self._h, int(on)))

    def stage_ms(self):
        """{S1..S5: ms} of the last profiled infer (waits for it to finish)."""
        ms = (C.c_float * 5)()
        self._check(lib().trk_profile_stage_ms(self._h, ms))
        return dict(zip(("s1_embed", "s2_frnn", "s3_filter", "s4_gnn", "s5_cc"), [float(v) for v in ms]))

    def kernel_ms(self):
        """(per-launch ms of the S3 hidden-layer GEMMs of the last profiled infer, rows per launch)."""
        n, rows = C.c_int32(0), C.c_int64(0)
        self._check(lib().trk_profile_kernel_ms(self._h, None, 0, C.byref(n), C.byref(rows)))
        ms = (C.c_float * max(1, n.value))()
        self._check(lib().trk_profile_kernel_ms(self._h, ms, n.value, C.byref(n), C.byref(rows)))
        return [float(ms[i]) for i in range(n.value)], int(rows.value)

    # ---- the call
    def infer(self, hits, event_offsets, *, want_edges=False, want_cand=False, want_embedding=False, want_tracks=False, out=None,
              stream=None):
        """hits: CUDA fp32 [N,3]; event_offsets: host int32 [B+1].  Returns dict of CUDA tensors (no sync)."""
        import torch
        off = np.ascontiguousarray(event_offsets, dtype=np.int32)
        n = int(off[-1]) if len(off) else 0
        dev = hits.device
        o = out if out is not None else {}
        if "labels" not in o:
            o["labels"] = torch.empty(n, dtype=torch.int32, device=dev)
            o["counts"] = torch.zeros(4, dtype=torch.int32, device=dev)
            if want_edges:
                cap = int(self.cfg.max_kept_edges)
                o["edge_src"] = torch.empty(cap, dtype=torch.int32, device=dev)
                o["edge_dst"] = torch.empty(cap, dtype=torch.int32, device=dev)
                o["edge_score"] = torch.empty(cap, dtype=torch.float32, device=dev)
            if want_cand:
                cap = int(self.cfg.max_cand_edges)
                o["cand_src"] = torch.empty(cap, dtype=torch.int32, device=dev)
                o["cand_dst"] = torch.empty(cap, dtype=torch.int32, device=dev)
                o["cand_score"] = torch.empty(cap, dtype=torch.float32, device=dev)
            if want_embedding:
                o["embedding"] = torch.empty(n, self.d_e, dtype=torch.float32, device=dev)
            if want_tracks:
                o["track_offsets"] = torch.zeros(max(n, 1) + 1, dtype=torch.int32, device=dev)
                o["track_hits"] = torch.empty(n, dtype=torch.int32, device=dev)
                o["track_counts"] = torch.zeros(2, dtype=torch.int32, device=dev)
        b = TrkBatch(len(off) - 1, off.ctypes.data_as(_i32p), _ptr(hits))
        r = TrkResult()
        r.labels, r.counts = _ptr(o["labels"]), _ptr(o["counts"])
        r.edge_src, r.edge_dst, r.edge_score = _ptr(o.get("edge_src")), _ptr(o.get("edge_dst")), _ptr(o.get("edge_score"))
        r.edge_capacity = o["edge_src"].numel() if "edge_src" in o else 0
        r.cand_src, r.cand_dst, r.cand_score = _ptr(o.get("cand_src")), _ptr(o.get("cand_dst")), _ptr(o.get("cand_score"))
        r.cand_capacity = o["cand_src"].numel() if "cand_src" in o else 0
        r.embedding = _ptr(o.get("embedding"))
        r.track_offsets, r.track_hits, r.track_counts = _ptr(o.get("track_offsets")), _ptr(o.get("track_hits")), _ptr(o.get("track_counts"))
        r.track_capacity = o["track_offsets"].numel() - 1 if "track_offsets" in o else 0
        self._check(lib().trk_infer(self._h, C.byref(b), C.byref(r), _stream_ptr(stream)))
        return o

    def infer_host(self, hits_host, event_offsets, labels_host=None, counts_host=None):
        """HOST buffers in, HOST labels out (H2D + pipeline + D2H + sync inside the call)."""
        off = np.ascontiguousarray(event_offsets, dtype=np.int32)
        n = int(off[-1])
        if labels_host is None:
            labels_host = np.empty(n, dtype=np.int32)
        if counts_host is None:
            counts_host = np.zeros(4, dtype=np.int32)

        def hp(a):
            return C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data)
        self._check(lib().trk_infer_host(self._h, len(off) - 1, off.ctypes.data_as(_i32p), hp(hits_host), hp(labels_host), hp(counts_host)))
        return labels_host, counts_host

    def infer_host_tracks(self, hits_host, event_offsets, labels_host=None):
        """HOST hits in, HOST track candidates out: (track_offsets [T+1], track_hits, labels, counts [6])."""
        off = np.ascontiguousarray(event_offsets, dtype=np.int32)
        n = int(off[-1])
        if labels_host is None:
            labels_host = np.empty(n, dtype=np.int32)
        toff = np.zeros(n + 1, dtype=np.int32)
        thit = np.empty(n, dtype=np.int32)
        counts = np.zeros(6, dtype=np.int32)

        def hp(a):
            return C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data)
        self._check(lib().trk_infer_host_tracks(self._h, len(off) - 1, off.ctypes.data_as(_i32p), hp(hits_host), hp(labels_host), hp(toff),
                                                hp(thit), hp(counts)))
        return toff[:counts[4] + 1], thit[:counts[5]], labels_host, counts

    # ---- stage hooks (device tensors in, device tensors out, enqueued on the current stream)
    def stage_embed(self, hits, stream=None):
        import torch
        n = hits.shape[0]
        emb = torch.empty(n, self.d_e, dtype=torch.float32, device=hits.device)
        self._check(lib().trk_stage_embed(self._h, _ptr(hits), n, _ptr(emb), _stream_ptr(stream)))
        return emb

    def stage_frnn(self, emb, hits, event_offsets, capacity=None, stream=None):
        import torch
        off = np.ascontiguousarray(event_offsets, dtype=np.int32)
        n = int(off[-1])
        cap = int(capacity if capacity is not None else min(int(self.cfg.max_cand_edges), max(1, n) * self.cfg.frnn_k))
        dev = hits.device
        src = torch.empty(cap, dtype=torch.int32, device=dev)
        dst = torch.empty(cap, dtype=torch.int32, device=dev)
        rowptr = torch.zeros(n + 1, dtype=torch.int32, device=dev)
        count = torch.zeros(2, dtype=torch.int32, device=dev)
        self._check(lib().trk_stage_frnn(self._h, _ptr(emb), _ptr(hits), off.ctypes.data_as(_i32p), len(off) - 1, _ptr(src), _ptr(dst),
                                         _ptr(rowptr), cap, _ptr(count), _stream_ptr(stream)))
        return src, dst, rowptr, count

    def stage_filter(self, feat, src, dst, stream=None):
        import torch
        score = torch.empty(src.numel(), dtype=torch.float32, device=src.device)
        self._check(lib().trk_stage_filter(self._h, _ptr(feat), feat.shape[0], _ptr(src), _ptr(dst), src.numel(), _ptr(score),
                                           _stream_ptr(stream)))
        return score

    def stage_compact(self, src, dst, score, capacity=None, stream=None):
        import torch
        cap = int(capacity if capacity is not None else max(1, src.numel()))
        os_ = torch.empty(cap, dtype=torch.int32, device=src.device)
        od = torch.empty(cap, dtype=torch.int32, device=src.device)
        count = torch.zeros(2, dtype=torch.int32, device=src.device)
        self._check(lib().trk_stage_compact(self._h, _ptr(src), _ptr(dst), _ptr(score), src.numel(), _ptr(os_), _ptr(od), cap,
                                            _ptr(count), _stream_ptr(stream)))
        return os_, od, count

    def stage_gnn(self, hits, src, dst, stream=None):
        import torch
        score = torch.empty(src.numel(), dtype=torch.float32, device=hits.device)
        self._check(lib().trk_stage_gnn(self._h, _ptr(hits), hits.shape[0], _ptr(src), _ptr(dst), src.numel(), _ptr(score),
                                        _stream_ptr(stream)))
        return score

    def stage_gnn_csr(self, hits, src, dst, stream=None):
        """The S4 scatter structure: (in_rowptr [n+1], in_perm [n_edges], out_rowptr [n+1])."""
        import torch
        n = hits.shape[0]
        in_rowptr = torch.empty(n + 1, dtype=torch.int32, device=hits.device)
        out_rowptr = torch.empty(n + 1, dtype=torch.int32, device=hits.device)
        in_perm = torch.empty(src.numel(), dtype=torch.int32, device=hits.device)
        self._check(lib().trk_stage_gnn_csr(self._h, _ptr(hits), n, _ptr(src), _ptr(dst), src.numel(), _ptr(in_rowptr), _ptr(in_perm),
                                            _ptr(out_rowptr), _stream_ptr(stream)))
        return in_rowptr, in_perm, out_rowptr

    def stage_cc(self, n, src, dst, score, cut, stream=None):
        import torch
        labels = torch.empty(n, dtype=torch.int32, device=src.device)
        self._check(lib().trk_stage_cc(self._h, n, _ptr(src), _ptr(dst), _ptr(score), src.numel(), float(cut), _ptr(labels),
                                       _stream_ptr(stream)))
        return labels


    def stage_tracks(self, labels, min_hits, capacity=None, stream=None):
        """labels CUDA int32 [n] -> (track_offsets [capacity+1], track_hits [n], track_counts [3] = {T, hits, overflow})."""
        import torch
        n = labels.numel()
        cap = int(capacity if capacity is not None else max(n, 1))
        toff = torch.zeros(cap + 1, dtype=torch.int32, device=labels.device)
        thit = torch.empty(n, dtype=torch.int32, device=labels.device)
        cnt = torch.zeros(3, dtype=torch.int32, device=labels.device)
        self._check(lib().trk_stage_tracks(self._h, _ptr(labels), n, int(min_hits), _ptr(toff), cap, _ptr(thit), _ptr(cnt),
                                           _stream_ptr(stream)))
        return toff, thit, cnt


def gemm_bf16(a, w, bias, relu=True, pair=True, stream=None):
    """out = act(a @ w.T + bias) on the tcgen05 GEMM kernel; a [m,k] bf16, w [n,k] bf16, bias fp32 [n]."""
    import torch
    m, k = a.shape
    n = w.shape[0]
    out = torch.empty(m, n, dtype=torch.bfloat16, device=a.device)
    st = lib().trk_gemm_bf16(_ptr(a), _ptr(w), _ptr(bias), _ptr(out), m, n, k, int(relu), int(bool(pair)), _stream_ptr(stream))
    if st != 0:
        raise TrkError(st, lib().trk_last_error(None).decode())
    return out


def cc_noalloc(n, src, dst, score, cut, labels, stream=None):
    """trk_cc_noalloc: S5 labels for callers that must not allocate device memory (a backend inside a fixed memory budget,
    code where cudaMalloc is forbidden or stalls the device).  No context: the union-find scratch is a fixed array inside
    libtrk.so, so n <= CC_NOALLOC_MAX_HITS.  `labels` (CUDA int32 [n]) is the caller's buffer and is written in place --
    this wrapper allocates nothing either.  Runs on the current device; calls that overlap on one GPU race on the scratch."""
    st = lib().trk_cc_noalloc(int(n), _ptr(src), _ptr(dst), _ptr(score), 0 if src is None else src.numel(), float(cut), _ptr(labels),
                              _stream_ptr(stream))
    if st != 0:
        raise TrkError(st, lib().trk_last_error(None).decode())
    return labels
