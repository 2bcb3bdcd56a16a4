"""Thin ctypes binding of liblsa (include/lsa.h): argument marshalling only.

Every step of the LSA path runs in the CUDA kernels behind the C ABI; PyTorch is used here
for device / pinned-host memory and streams.  There is no CPU fallback: importing this
module without the built library raises, and so does calling it without a CUDA device.

Functions mirror the C names: lsa_init_pools, lsa_index_select, lsa_fetch_chunks,
lsa_decode_attention, lsa_step (+ support calls).  `LsaContext` owns the opaque handle and
keeps the caller's tensors alive for the lifetime of the context (the library never copies
them).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence, Tuple

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblsa.so")

LSA_F32, LSA_BF16 = 0, 1
LSA_ATTN_AUTO, LSA_ATTN_SIMT, LSA_ATTN_TCGEN05 = 0, 1, 2
LSA_MERGE_AUTO, LSA_MERGE_KERNEL, LSA_MERGE_FUSED = 0, 1, 2
LSA_COLD_NATIVE, LSA_COLD_FP8_E4M3 = 0, 1
LSA_INDEXER_DUAL_ENCODER, LSA_INDEXER_LEVEL1 = 0, 1

STATUS = {0: "LSA_OK", -1: "LSA_ERR_INVALID_ARG", -2: "LSA_ERR_CUDA", -3: "LSA_ERR_POOL_EXHAUSTED",
          -4: "LSA_ERR_OOM", -5: "LSA_ERR_STATE", -6: "LSA_ERR_UNSUPPORTED"}

EXPORTS = ["lsa_init_pools", "lsa_index_select", "lsa_fetch_chunks", "lsa_commit_tables",
           "lsa_decode_attention", "lsa_step", "lsa_step_host", "lsa_step_host_async", "lsa_host_wait", "lsa_set_chunk_emb",
           "lsa_get_page_table", "lsa_get_residency", "lsa_get_stats", "lsa_get_step", "lsa_sync",
           "lsa_profile_enable", "lsa_profile_read", "lsa_timeline_enable", "lsa_timeline_read", "lsa_l1_init", "lsa_l1_select", "lsa_set_indexer",
           "lsa_l2_init", "lsa_l2_select", "lsa_step_l2", "lsa_l2_get_mask", "lsa_step_graph", "lsa_graph_stats", "lsa_export_chunks",
           "lsa_append_compressed", "lsa_index_select_static", "lsa_last_error", "lsa_destroy", "lsa_version"]


class LsaError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


class lsa_config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("dtype", C.c_int32), ("B", C.c_int32), ("H", C.c_int32),
                ("D", C.c_int32), ("C", C.c_int32), ("W", C.c_int32), ("Dh", C.c_int32), ("E", C.c_int32),
                ("k", C.c_int32), ("tau", C.c_int32), ("recall_lag", C.c_int32), ("sm_scale", C.c_float),
                ("hot_pages", C.c_int64), ("hot_pool", C.c_void_p), ("W_q", C.c_void_p),
                ("stream_compute", C.c_void_p), ("stream_fetch", C.c_void_p), ("attn_impl", C.c_int32),
                ("step_overlap", C.c_int32), ("max_ctas", C.c_int32), ("merge_mode", C.c_int32),
                ("cold_format", C.c_int32), ("reserved0", C.c_int32)]


class lsa_seq_desc(C.Structure):
    _fields_ = [("cold_csa", C.c_void_p), ("n_csa", C.c_int64), ("chunk_emb", C.c_void_p),
                ("hca_k", C.c_void_p), ("hca_v", C.c_void_p), ("n_hca", C.c_int64), ("win_k", C.c_void_p),
                ("win_v", C.c_void_p), ("w_len", C.c_int32), ("w_head", C.c_int32), ("step0", C.c_int64),
                ("cap_csa", C.c_int64), ("cap_hca", C.c_int64), ("cold_scale", C.c_void_p)]


class lsa_stats(C.Structure):
    _fields_ = [("triggers", C.c_uint64), ("hits", C.c_uint64), ("misses", C.c_uint64),
                ("evictions", C.c_uint64), ("bytes_fetched", C.c_uint64), ("steps", C.c_uint64),
                ("attn_launches", C.c_uint64), ("index_launches", C.c_uint64), ("pool_error", C.c_int32),
                ("attn_impl", C.c_int32), ("attn_ctas", C.c_int32), ("reserved", C.c_int32),
                ("csa_appended", C.c_uint64), ("hca_appended", C.c_uint64), ("chunks_exported", C.c_uint64)]


class lsa_l1_layer(C.Structure):
    _fields_ = [("W_dq", C.c_void_p), ("W_iuq", C.c_void_p), ("W_w", C.c_void_p)]


class lsa_l2_config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("c_I", C.c_int32), ("n_h", C.c_int32), ("k2", C.c_int32)]


class lsa_l1_config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_layers", C.c_int32), ("d_c", C.c_int32), ("c_I", C.c_int32),
                ("n_h", C.c_int32), ("threshold", C.c_float), ("layers", lsa_l1_layer * 4)]


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2606_09079_b200.build` "
            "(or __graft_entry__.build()).  There is no CPU fallback for the LSA path.")
    lib = C.CDLL(LIB_PATH)
    vp, i32p, f32p = C.c_void_p, C.POINTER(C.c_int32), C.c_void_p
    lib.lsa_init_pools.argtypes = [C.POINTER(lsa_config), C.POINTER(lsa_seq_desc), C.POINTER(vp)]
    lib.lsa_index_select.argtypes = [vp, vp, i32p, C.c_int32, vp, f32p]
    lib.lsa_fetch_chunks.argtypes = [vp, i32p, C.c_int32, vp]
    lib.lsa_commit_tables.argtypes = [vp]
    lib.lsa_decode_attention.argtypes = [vp, vp, vp, f32p]
    lib.lsa_step.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.lsa_step_host.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.lsa_step_host_async.argtypes = [vp, vp, vp, vp, vp, vp, C.POINTER(C.c_uint64)]
    lib.lsa_host_wait.argtypes = [vp, C.c_uint64]
    lib.lsa_set_chunk_emb.argtypes = [vp, C.c_int32, vp]
    lib.lsa_get_page_table.argtypes = [vp, C.c_int32, C.c_int32, i32p, i32p, i32p]
    lib.lsa_get_residency.argtypes = [vp, C.c_int32, i32p]
    lib.lsa_get_stats.argtypes = [vp, C.POINTER(lsa_stats)]
    lib.lsa_get_step.argtypes = [vp, C.c_int32, C.POINTER(C.c_int64)]
    lib.lsa_sync.argtypes = [vp]
    lib.lsa_profile_enable.argtypes = [vp, C.c_int32]
    lib.lsa_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    lib.lsa_timeline_enable.argtypes = [vp, C.c_int32]
    lib.lsa_timeline_read.argtypes = [vp, vp, C.POINTER(C.c_uint64)]
    lib.lsa_l1_init.argtypes = [vp, C.POINTER(lsa_l1_config), C.POINTER(vp)]
    lib.lsa_l1_select.argtypes = [vp, vp, i32p, C.c_int32, vp, f32p]
    lib.lsa_set_indexer.argtypes = [vp, C.c_int32]
    lib.lsa_l2_init.argtypes = [vp, C.POINTER(lsa_l2_config), C.POINTER(vp)]
    lib.lsa_l2_select.argtypes = [vp, vp, vp, vp, vp]
    lib.lsa_l2_get_mask.argtypes = [vp, C.c_int32, vp]
    lib.lsa_export_chunks.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, vp]
    lib.lsa_index_select_static.argtypes = [C.c_int32, vp, vp, C.POINTER(C.c_void_p), C.POINTER(C.c_int32), C.c_int32, C.c_int32,
                                            C.c_int32, C.c_int32, vp, vp, vp]
    lib.lsa_append_compressed.argtypes = [vp, C.POINTER(C.c_int32), C.c_int32, vp, vp, vp, vp, vp]
    lib.lsa_step_graph.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.lsa_graph_stats.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    lib.lsa_step_l2.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
    lib.lsa_last_error.argtypes = [vp]
    lib.lsa_last_error.restype = C.c_char_p
    lib.lsa_destroy.argtypes = [vp]
    lib.lsa_destroy.restype = None
    lib.lsa_version.argtypes = []
    for name in EXPORTS:
        if name not in ("lsa_last_error", "lsa_destroy"):
            getattr(lib, name).restype = C.c_int
    return lib


_lib = _load()


def _torch_dtype(dtype: int):
    return torch.float32 if dtype == LSA_F32 else torch.bfloat16


def _dev_ptr(t: Optional[torch.Tensor], dtype=None, what="tensor") -> Optional[int]:
    if t is None:
        return None
    if not t.is_cuda:
        raise LsaError(-1, f"{what} must be a CUDA tensor")
    if not t.is_contiguous():
        raise LsaError(-1, f"{what} must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise LsaError(-1, f"{what} must have dtype {dtype}, got {t.dtype}")
    return t.data_ptr()


def _host_ptr(t: Optional[torch.Tensor], dtype=None, what="tensor") -> Optional[int]:
    if t is None:
        return None
    if t.is_cuda or not t.is_contiguous():
        raise LsaError(-1, f"{what} must be a contiguous host tensor")
    if dtype is not None and t.dtype != dtype:
        raise LsaError(-1, f"{what} must have dtype {dtype}, got {t.dtype}")
    return t.data_ptr()


def _ids(seq_ids: Sequence[int]):
    arr = (C.c_int32 * len(seq_ids))(*[int(x) for x in seq_ids])
    return arr, len(seq_ids)


class LsaContext:
    """Owns one lsa_ctx.  See include/lsa.h for the meaning of every argument.

    Stream contract (include/lsa.h "Conventions"): results are written on the library's streams - `out` / `lse` on
    stream_compute, `sel_idx` / `sel_score` on stream_fetch - NOT on torch's current stream.  Tensors this wrapper
    allocates for them are marked with record_stream(), so the caching allocator cannot hand their memory out again
    while the library still writes it; a caller that reads them on another stream orders that stream behind the
    library's (ctx.stream_compute / ctx.stream_fetch, or ctx.sync())."""

    def _on(self, t, stream):
        if t is not None:
            t.record_stream(stream)
        return t

    def __init__(self, *, dtype: int, H: int, D: int, C_: int, W: int, Dh: int, E: int, k: int, tau: int,
                 hot_pool: torch.Tensor, W_q: torch.Tensor, seqs: Sequence[dict], recall_lag: int = 1,
                 sm_scale: float = 0.0, stream_compute: Optional[torch.cuda.Stream] = None,
                 stream_fetch: Optional[torch.cuda.Stream] = None, attn_impl: int = LSA_ATTN_AUTO,
                 step_overlap: int = 0, max_ctas: int = 0, merge_mode: int = LSA_MERGE_AUTO, cold_format: int = 0):
        if not torch.cuda.is_available():
            raise LsaError(-2, "no CUDA device: the LSA path has no CPU fallback")
        td = _torch_dtype(dtype)
        self.dtype, self.tdtype = dtype, td
        self.B, self.H, self.D, self.C, self.W, self.Dh, self.E, self.k, self.tau = len(seqs), H, D, C_, W, Dh, E, k, tau
        self.stream_compute = stream_compute or torch.cuda.Stream()
        self.stream_fetch = stream_fetch or torch.cuda.Stream()
        self._keep = [hot_pool, W_q, list(seqs)]
        page_elems = 2 * C_ * D
        if hot_pool.numel() % page_elems:
            raise LsaError(-1, "hot_pool size is not a whole number of pages")
        cfg = lsa_config()
        cfg.struct_size = C.sizeof(lsa_config)
        cfg.dtype, cfg.B, cfg.H, cfg.D, cfg.C, cfg.W = dtype, self.B, H, D, C_, W
        cfg.Dh, cfg.E, cfg.k, cfg.tau, cfg.recall_lag, cfg.sm_scale = Dh, E, k, tau, recall_lag, sm_scale
        cfg.hot_pages = hot_pool.numel() // page_elems
        cfg.hot_pool = _dev_ptr(hot_pool, td, "hot_pool")
        cfg.W_q = _dev_ptr(W_q, td, "W_q")
        cfg.stream_compute = self.stream_compute.cuda_stream
        cfg.stream_fetch = self.stream_fetch.cuda_stream
        cfg.attn_impl, cfg.step_overlap, cfg.max_ctas, cfg.merge_mode = attn_impl, step_overlap, max_ctas, merge_mode
        cfg.cold_format = cold_format
        descs = (lsa_seq_desc * self.B)()
        for b, s in enumerate(seqs):
            d = descs[b]
            cold = s.get("cold_csa")
            if cold is not None and not cold.is_pinned():
                raise LsaError(-1, f"seq {b}: cold_csa must be pinned host memory")
            d.cold_csa = _host_ptr(cold, torch.uint8 if cold_format == LSA_COLD_FP8_E4M3 else td, "cold_csa")
            d.cold_scale = _dev_ptr(s.get("cold_scale"), torch.float32, "cold_scale")
            d.n_csa = int(s["n_csa"])
            d.chunk_emb = _dev_ptr(s.get("chunk_emb"), td, "chunk_emb")
            d.hca_k = _dev_ptr(s.get("hca_k"), td, "hca_k")
            d.hca_v = _dev_ptr(s.get("hca_v"), td, "hca_v")
            d.n_hca = int(s["n_hca"]) if "n_hca" in s else (0 if s.get("hca_k") is None else s["hca_k"].shape[0])
            d.win_k = _dev_ptr(s.get("win_k"), td, "win_k")
            d.win_v = _dev_ptr(s.get("win_v"), td, "win_v")
            d.w_len = int(s.get("w_len", 0))
            d.w_head = int(s.get("w_head", 0))
            d.step0 = int(s.get("step0", 0))
            d.cap_csa = int(s.get("cap_csa", 0))
            d.cap_hca = int(s.get("cap_hca", 0))
        handle = C.c_void_p()
        rc = _lib.lsa_init_pools(C.byref(cfg), descs, C.byref(handle))
        if rc != 0:
            raise LsaError(rc, (_lib.lsa_last_error(None) or b"").decode())
        self._h = handle
        self.hot_pages = int(cfg.hot_pages)

    # -- helpers ---------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != 0:
            raise LsaError(rc, (_lib.lsa_last_error(self._h) or b"").decode())

    def close(self):
        if getattr(self, "_h", None):
            _lib.lsa_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the five path calls ---------------------------------------------------------------
    def index_select(self, h: torch.Tensor, seq_ids: Sequence[int], want_scores: bool = True):
        arr, n = _ids(seq_ids)
        sel = torch.empty((n, self.k), dtype=torch.int32, device=h.device)
        sc = torch.empty((n, self.k), dtype=torch.float32, device=h.device) if want_scores else None
        self._check(_lib.lsa_index_select(self._h, _dev_ptr(h, self.tdtype, "h"), arr, n, sel.data_ptr(),
                                          None if sc is None else sc.data_ptr()))
        return self._on(sel, self.stream_fetch), self._on(sc, self.stream_fetch)

    def l1_init(self, layers: Sequence[dict], index_k: Sequence[Sequence[torch.Tensor]], d_c: int, c_I: int = 128,
                n_h: int = 64, threshold: float = 0.5):
        """Paper-exact Level-1 indexer (Eq. 1-5, 13).  layers[l] = dict(W_dq [d_c][Dh], W_iuq [n_h*c_I][d_c],
        W_w [n_h][Dh]) bf16 CUDA tensors; index_k[b][l] = [n_csa_b][c_I] bf16 CUDA tensor."""
        cfg = lsa_l1_config()
        cfg.struct_size = C.sizeof(lsa_l1_config)
        cfg.n_layers, cfg.d_c, cfg.c_I, cfg.n_h, cfg.threshold = len(layers), d_c, c_I, n_h, threshold
        for l, lay in enumerate(layers):
            cfg.layers[l].W_dq = _dev_ptr(lay["W_dq"], self.tdtype, "W_dq")
            cfg.layers[l].W_iuq = _dev_ptr(lay["W_iuq"], self.tdtype, "W_iuq")
            cfg.layers[l].W_w = _dev_ptr(lay["W_w"], self.tdtype, "W_w")
        L = len(layers)
        ptrs = (C.c_void_p * (self.B * L))()
        for b in range(self.B):
            for l in range(L):
                t = index_k[b][l]
                ptrs[b * L + l] = _dev_ptr(t, self.tdtype, "index_k") if t is not None and t.numel() else None
        self._keep += [list(layers), [list(x) for x in index_k]]
        self._check(_lib.lsa_l1_init(self._h, C.byref(cfg), ptrs))

    def l2_init(self, index_k: Sequence[torch.Tensor], k2: int, c_I: int = 128, n_h: int = 64):
        """Level 2 (Eq. 6): index_k[b] = [n_csa_b][c_I] bf16 CUDA tensor of this layer's compressed indexer keys."""
        cfg = lsa_l2_config()
        cfg.struct_size = C.sizeof(lsa_l2_config)
        cfg.c_I, cfg.n_h, cfg.k2 = c_I, n_h, k2
        ptrs = (C.c_void_p * self.B)()
        for b in range(self.B):
            t = index_k[b]
            ptrs[b] = _dev_ptr(t, self.tdtype, "index_k") if t is not None and t.numel() else None
        self._keep += [list(index_k)]
        self._check(_lib.lsa_l2_init(self._h, C.byref(cfg), ptrs))
        self.k2 = k2

    def l2_select(self, q_idx: torch.Tensor, w_idx: torch.Tensor, want_entries: bool = True):
        sel = torch.empty((self.B, self.k2), dtype=torch.int32, device=q_idx.device) if want_entries else None
        sc = torch.empty((self.B, self.k2), dtype=torch.float32, device=q_idx.device) if want_entries else None
        self._check(_lib.lsa_l2_select(self._h, _dev_ptr(q_idx, self.tdtype, "q_idx"), _dev_ptr(w_idx, torch.float32, "w_idx"),
                                       None if sel is None else sel.data_ptr(), None if sc is None else sc.data_ptr()))
        return self._on(sel, self.stream_compute), self._on(sc, self.stream_compute)

    def l2_mask(self, seq: int):
        """Blocking: the row mask of the last Level-2 selection, as a bool array [k][C = 128]."""
        import numpy as np
        words = np.zeros(self.k * 4, dtype=np.uint32)
        self._check(_lib.lsa_l2_get_mask(self._h, seq, words.ctypes.data))
        bits = (words[:, None] >> np.arange(32, dtype=np.uint32)[None, :]) & 1
        return bits.reshape(self.k, 128).astype(bool)

    def step_l2(self, q, h, k_new, v_new, q_idx, w_idx, out=None):
        out = self._on(torch.empty_like(q), self.stream_compute) if out is None else out
        self._check(_lib.lsa_step_l2(self._h, _dev_ptr(q, self.tdtype, "q"), _dev_ptr(h, self.tdtype, "h"),
                                     _dev_ptr(k_new, self.tdtype, "k_new"), _dev_ptr(v_new, self.tdtype, "v_new"),
                                     _dev_ptr(q_idx, self.tdtype, "q_idx"), _dev_ptr(w_idx, torch.float32, "w_idx"),
                                     _dev_ptr(out, self.tdtype, "out")))
        return out

    def set_indexer(self, indexer: int):
        self._check(_lib.lsa_set_indexer(self._h, indexer))

    def l1_select(self, h: torch.Tensor, seq_ids: Sequence[int], want_scores: bool = True):
        arr, n = _ids(seq_ids)
        sel = torch.empty((n, self.k), dtype=torch.int32, device=h.device)
        sc = torch.empty((n, self.k), dtype=torch.float32, device=h.device) if want_scores else None
        self._check(_lib.lsa_l1_select(self._h, _dev_ptr(h, self.tdtype, "h"), arr, n, sel.data_ptr(),
                                       None if sc is None else sc.data_ptr()))
        return self._on(sel, self.stream_fetch), self._on(sc, self.stream_fetch)

    def fetch_chunks(self, seq_ids: Sequence[int], sel_idx: torch.Tensor):
        arr, n = _ids(seq_ids)
        self._check(_lib.lsa_fetch_chunks(self._h, arr, n, _dev_ptr(sel_idx, torch.int32, "sel_idx")))

    def commit_tables(self):
        self._check(_lib.lsa_commit_tables(self._h))

    def decode_attention(self, q: torch.Tensor, out: Optional[torch.Tensor] = None, want_lse: bool = False):
        out = self._on(torch.empty_like(q), self.stream_compute) if out is None else out
        lse = self._on(torch.empty((self.B, self.H), dtype=torch.float32, device=q.device), self.stream_compute) if want_lse else None
        self._check(_lib.lsa_decode_attention(self._h, _dev_ptr(q, self.tdtype, "q"), _dev_ptr(out, self.tdtype, "out"),
                                              None if lse is None else lse.data_ptr()))
        return (out, lse) if want_lse else out

    def step(self, q, h, k_new=None, v_new=None, out=None):
        out = self._on(torch.empty_like(q), self.stream_compute) if out is None else out
        self._check(_lib.lsa_step(self._h, _dev_ptr(q, self.tdtype, "q"), _dev_ptr(h, self.tdtype, "h"),
                                  _dev_ptr(k_new, self.tdtype, "k_new"), _dev_ptr(v_new, self.tdtype, "v_new"),
                                  _dev_ptr(out, self.tdtype, "out")))
        return out

    def bind_step(self, q, h, k_new, v_new, out):
        """lsa_step on fixed buffers: the arguments are checked and converted once, the returned callable only makes the
        C call (a decode loop that reuses its buffers pays the marshalling once instead of every step)."""
        args = (self._h, C.c_void_p(_dev_ptr(q, self.tdtype, "q")), C.c_void_p(_dev_ptr(h, self.tdtype, "h")),
                C.c_void_p(_dev_ptr(k_new, self.tdtype, "k_new")), C.c_void_p(_dev_ptr(v_new, self.tdtype, "v_new")),
                C.c_void_p(_dev_ptr(out, self.tdtype, "out")))
        keep = (q, h, k_new, v_new, out)
        fn, check = _lib.lsa_step, self._check

        def call(_keep=keep):
            rc = fn(*args)
            if rc:
                check(rc)
        return call

    def export_chunks(self, seq: int, first_chunk: int, src: torch.Tensor):
        """KV export (VRAM -> pinned cold pool): src = [n][2][C][D] CUDA tensor of page images for chunks first_chunk.."""
        self._check(_lib.lsa_export_chunks(self._h, seq, first_chunk, int(src.shape[0]), _dev_ptr(src, self.tdtype, "src")))

    def append_compressed(self, seq_ids: Sequence[int], csa_k=None, csa_v=None, hca_k=None, hca_v=None, emb_rows=None):
        """Hand over the compressed entries of the tokens decoded since the last call (NEXT-4): csa_k / csa_v [n][D],
        hca_k / hca_v [n][D], emb_rows [n][E] CUDA tensors (row i belongs to seq_ids[i])."""
        arr, n = _ids(seq_ids)
        self._check(_lib.lsa_append_compressed(self._h, arr, n, _dev_ptr(csa_k, self.tdtype, "csa_k"), _dev_ptr(csa_v, self.tdtype, "csa_v"),
                                               _dev_ptr(hca_k, self.tdtype, "hca_k"), _dev_ptr(hca_v, self.tdtype, "hca_v"),
                                               _dev_ptr(emb_rows, self.tdtype, "emb_rows")))
        for t in (csa_k, csa_v, hca_k, hca_v, emb_rows):
            self._on(t, self.stream_compute)

    def step_graph(self, q, h, k_new=None, v_new=None, out=None):
        """lsa_step with the non-trigger step replayed from a CUDA graph (keep q / k_new / v_new / out at fixed addresses)."""
        out = self._on(torch.empty_like(q), self.stream_compute) if out is None else out
        self._check(_lib.lsa_step_graph(self._h, _dev_ptr(q, self.tdtype, "q"), _dev_ptr(h, self.tdtype, "h"),
                                        _dev_ptr(k_new, self.tdtype, "k_new"), _dev_ptr(v_new, self.tdtype, "v_new"),
                                        _dev_ptr(out, self.tdtype, "out")))
        return out

    def graph_stats(self):
        cap, rep = C.c_uint64(0), C.c_uint64(0)
        self._check(_lib.lsa_graph_stats(self._h, C.byref(cap), C.byref(rep)))
        return dict(captures=cap.value, replays=rep.value)

    def step_host(self, q, h, k_new, v_new, out):
        self._check(_lib.lsa_step_host(self._h, _host_ptr(q, self.tdtype, "q"), _host_ptr(h, self.tdtype, "h"),
                                       _host_ptr(k_new, self.tdtype, "k_new"), _host_ptr(v_new, self.tdtype, "v_new"),
                                       _host_ptr(out, self.tdtype, "out")))
        return out

    def step_host_async(self, q, h, k_new, v_new, out) -> int:
        """lsa_step_host without the wait; returns the ticket for host_wait (buffers must stay untouched until then)."""
        t = C.c_uint64(0)
        self._check(_lib.lsa_step_host_async(self._h, _host_ptr(q, self.tdtype, "q"), _host_ptr(h, self.tdtype, "h"),
                                             _host_ptr(k_new, self.tdtype, "k_new"), _host_ptr(v_new, self.tdtype, "v_new"),
                                             _host_ptr(out, self.tdtype, "out"), C.byref(t)))
        return t.value

    def host_wait(self, ticket: int):
        self._check(_lib.lsa_host_wait(self._h, ticket))

    # -- support -----------------------------------------------------------------------------
    def set_chunk_emb(self, seq: int, emb: torch.Tensor):
        self._keep.append(emb)
        self._check(_lib.lsa_set_chunk_emb(self._h, seq, _dev_ptr(emb, self.tdtype, "chunk_emb")))

    def page_table(self, seq: int, which: int = 0) -> Tuple[List[int], List[int]]:
        ch, pg, n = (C.c_int32 * self.k)(), (C.c_int32 * self.k)(), C.c_int32(0)
        self._check(_lib.lsa_get_page_table(self._h, seq, which, ch, pg, C.byref(n)))
        return list(ch[: n.value]), list(pg[: n.value])

    def residency(self, seq: int, n_chunks: int) -> List[int]:
        buf = (C.c_int32 * max(n_chunks, 1))()
        self._check(_lib.lsa_get_residency(self._h, seq, buf))
        return list(buf[:n_chunks])

    def stats(self) -> dict:
        st = lsa_stats()
        self._check(_lib.lsa_get_stats(self._h, C.byref(st)))
        return {f: getattr(st, f) for f, _ in lsa_stats._fields_ if f != "reserved"}

    def get_step(self, seq: int) -> int:
        v = C.c_int64(0)
        self._check(_lib.lsa_get_step(self._h, seq, C.byref(v)))
        return v.value

    def sync(self):
        self._check(_lib.lsa_sync(self._h))

    PHASES = ("prestep", "attention", "combine", "index", "residency", "fetch", "attention_dev")

    def profile_enable(self, capacity: int):
        self._check(_lib.lsa_profile_enable(self._h, capacity))

    TL_SHAPE = (16, 160, 12)      # LSA_TL_LAUNCHES, LSA_TL_CTAS, LSA_TL_EVENTS
    TL_EVENTS = ("entry", "setup", "first_s", "last_pv", "epilogue", "arrived", "all_arrived", "merged", "exit", "smid", "n_ctas", "seq")

    def timeline_enable(self, on: bool = True):
        self._check(_lib.lsa_timeline_enable(self._h, 1 if on else 0))

    def timeline_read(self):
        """(uint64 array [launch record][CTA][event] of %globaltimer nanoseconds, launches stamped so far); include/lsa.h LSA_TL_*"""
        import numpy as np
        buf = np.zeros(self.TL_SHAPE, dtype=np.uint64)
        n = C.c_uint64(0)
        self._check(_lib.lsa_timeline_read(self._h, buf.ctypes.data_as(C.c_void_p), C.byref(n)))
        return buf, int(n.value)

    def profile_read(self) -> dict:
        ms, cnt = (C.c_double * 7)(), (C.c_int64 * 7)()
        self._check(_lib.lsa_profile_read(self._h, ms, cnt))
        return {p: dict(ms=ms[i], count=cnt[i]) for i, p in enumerate(self.PHASES)}


# C-named free functions (same names as the ABI) --------------------------------------------------
def lsa_init_pools(**kw) -> LsaContext:
    return LsaContext(**kw)


def lsa_index_select(ctx: LsaContext, h, seq_ids, want_scores=True):
    return ctx.index_select(h, seq_ids, want_scores)


def lsa_fetch_chunks(ctx: LsaContext, seq_ids, sel_idx):
    return ctx.fetch_chunks(seq_ids, sel_idx)


def lsa_decode_attention(ctx: LsaContext, q, out=None, want_lse=False):
    return ctx.decode_attention(q, out, want_lse)


def lsa_step(ctx: LsaContext, q, h, k_new=None, v_new=None, out=None):
    return ctx.step(q, h, k_new, v_new, out)


def index_select_static(dtype: int, W_q: torch.Tensor, h: torch.Tensor, chunk_emb: Sequence[torch.Tensor], k: int,
                        sel_idx: torch.Tensor, sel_score: Optional[torch.Tensor] = None,
                        stream: Optional[torch.cuda.Stream] = None) -> None:
    """lsa_index_select_static: S1-S3 with the library's static device scratch - allocates nothing (see include/lsa.h for
    the limits and the no-overlap rule).  h [n][Dh], chunk_emb: n tensors [n_chunks_i][E], sel_idx [n][k] int32 and
    sel_score [n][k] fp32 are the CALLER's CUDA tensors; the kernels run on `stream` (default: torch's current stream)."""
    td = _torch_dtype(dtype)
    n = len(chunk_emb)
    if h.dim() != 2 or h.shape[0] != n:
        raise LsaError(-1, "h must be [n][Dh] with one row per embedding table")
    if sel_idx.dtype != torch.int32 or tuple(sel_idx.shape) != (n, k) or not sel_idx.is_cuda or not sel_idx.is_contiguous():
        raise LsaError(-1, "sel_idx must be a contiguous CUDA int32 tensor [n][k]")
    if sel_score is not None and (sel_score.dtype != torch.float32 or tuple(sel_score.shape) != (n, k) or not sel_score.is_cuda
                                  or not sel_score.is_contiguous()):
        raise LsaError(-1, "sel_score must be a contiguous CUDA float32 tensor [n][k]")
    E = int(W_q.shape[0])
    for e in chunk_emb:
        if e.dim() != 2 or int(e.shape[1]) != E:
            raise LsaError(-1, "every chunk_emb must be [n_chunks][E]")
    embs = (C.c_void_p * n)(*[_dev_ptr(e, td, "chunk_emb") for e in chunk_emb])
    ncs = (C.c_int32 * n)(*[int(e.shape[0]) for e in chunk_emb])
    st = torch.cuda.current_stream(h.device) if stream is None else stream
    with torch.cuda.device(h.device):
        rc = _lib.lsa_index_select_static(dtype, _dev_ptr(W_q, td, "W_q"), _dev_ptr(h, td, "h"), embs, ncs, n, E, int(W_q.shape[1]), k,
                                          sel_idx.data_ptr(), None if sel_score is None else sel_score.data_ptr(), st.cuda_stream)
    if rc != 0:
        raise LsaError(rc, (_lib.lsa_last_error(None) or b"").decode())


def lsa_version() -> int:
    return _lib.lsa_version()
