"""Glue shared by the tests: build the oracle (and, on a GPU, the CUDA context) from one
seeded workload.  Lives in tests/ because only tests may touch oracle/."""
from __future__ import annotations

import numpy as np

from oracle import LsaOracle
from paper_2606_09079_b200.workloads import LsaWorkload


def make_oracle(wl: LsaWorkload, trigger_idx: int = 0, **over) -> LsaOracle:
    c = wl.cfg
    kw = dict(
        dtype=c.dtype, H=c.H, D=c.D, C=c.C, W=c.W, k=c.k, tau=c.tau, recall_lag=c.recall_lag,
        hot_pages=c.hot_pages, W_q=wl.W_q, cold_csa=wl.cold_csa,
        n_csa=[c.n_csa(b) for b in range(c.B)],
        chunk_emb=[wl.chunk_emb(b, trigger_idx) for b in range(c.B)],
        hca_k=wl.hca_k, hca_v=wl.hca_v, win_k=wl.win_k, win_v=wl.win_v,
        w_len=[min(c.W, c.L[b]) for b in range(c.B)], w_head=[0] * c.B,
        step0=[c.step0(b) for b in range(c.B)])
    kw.update(over)
    return LsaOracle(**kw)


def apply_emb_updates(wl: LsaWorkload, oracle: LsaOracle, global_step: int, gpu_embs=None):
    """Needle drift (cfg 2-4): rewrite embedding rows before the trigger at `global_step`."""
    import torch
    from paper_2606_09079_b200.workloads import to_torch
    c = wl.cfg
    for b in range(c.B):
        if not wl.fires(b, global_step):
            continue
        upd = wl.emb_row_updates(b, wl.trigger_index(b, global_step))
        if upd is None:
            continue
        ids, rows = upd
        oracle.chunk_emb[b] = oracle.chunk_emb[b].copy()
        oracle.chunk_emb[b][ids] = rows
        if gpu_embs is not None:
            gpu_embs[b][torch.from_numpy(ids).to(gpu_embs[b].device)] = to_torch(rows, c.dtype).to(gpu_embs[b].device)
