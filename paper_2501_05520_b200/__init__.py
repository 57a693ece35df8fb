"""B200-native Exa.TrkX inference hot path (arXiv 2501.05520, section 2.2.2): Python binding of libtrk.so.

    from paper_2501_05520_b200 import Trk
The CUDA library is loaded lazily by `binding.lib()`; it is required -- there is no CPU fallback.
"""
from .binding import CC_NOALLOC_MAX_HITS, EXPORTS, LIB_PATH, Trk, TrkError, cc_noalloc, gemm_bf16, lib  # noqa: F401


def trk_from_config(cfg: dict, model: dict, calib: dict, *, max_hits: int, max_events: int = 1, max_cand_edges=None,
                    max_kept_edges=None, precision=None, use_grid_proj=True, gnn_layernorm=True, device=0, min_track_hits=3, filter_chunk_rows=0,
                    grid_max=0) -> "Trk":
    """Convenience: build a Trk from a plain config dict (keys as in synth.configs.CONFIGS) and a calibration dict."""
    return Trk(model=model, precision=precision or cfg["precision"], frnn_radius=calib["frnn_radius"], frnn_k=cfg["frnn_k"],
               filter_input=cfg["filter_input"], filter_cut=calib["filter_cut"], gnn_hidden=cfg["gnn_hidden"],
               gnn_iters=cfg["gnn_iters"], gnn_cut=cfg["gnn_cut"], max_hits=max_hits, max_events=max_events,
               max_cand_edges=max_cand_edges, max_kept_edges=max_kept_edges, gnn_layernorm=gnn_layernorm,
               grid_proj=calib.get("grid_proj") if use_grid_proj else None, device=device, min_track_hits=min_track_hits,
               filter_chunk_rows=filter_chunk_rows, grid_max=grid_max)
