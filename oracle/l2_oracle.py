"""CPU oracle for Level-2 of Lookahead Sparse Attention: the native Lightning Indexer restricted to the
resident recalled set, and core attention over its Top-k entries.

TEST INFRASTRUCTURE - NOT PRODUCT CODE (same rules as oracle/lsa_oracle.py: only tests/, smoke() and
bench.py's cpu_baseline legs may import it; it shares no code with the CUDA path).

Plain numpy, float64 from the STORED (bf16-rounded) inputs, in the paper's order (`P:n` = PAPER.md line n):

  P:75     "This Sigmoid activation stands as the only architectural departure from the native Lightning
           Indexer": the native score is Eq.(4) without the sigmoid,
               Score_native(i, s) = sum_h w_{i,h} ReLU( q_{i,h} . K_s^IComp )
  P:79-83  Eq.(6): once C_t^MemComp is resident, "the native Lightning Indexer calculates the token-level
           matching scores within this restricted C_t^MemComp boundary instead of scanning the full context
           ... to select the final fine-grained Top-k core compressed entries"
               C_i^CoreComp = { C_s in C_t^MemComp | Score_native(i, s) in Top-k }
  P:85     "The selected C_i^CoreComp entries are then concatenated with the non-offloadable sliding window KV
           cache to participate in the final core attention computation"  (+ all HCA entries: BASELINE.json
           north_star, DESIGN R5)
  P:187    in-graph ops "read residency bitmap, mask, Top-k, remap, MQA": it runs EVERY decode step i.

Readings:
  M1  C_t^MemComp = the valid rows of the pages of the sequence's CURRENT page table (what Level 1 recalled
      and S6 made visible); rows past n_csa in a partial last chunk are not entries.
  M2  Top-k = the first min(k2, |C_t^MemComp|) entries by (score descending, entry id ascending), entry id
      s = chunk * C + row (the paper gives no tie rule; same rule as BASELINE.json's top-k).
  M3  q_{i,h} and w_{i,h} of decode token i are inputs, as the attention query q is (the projections that make
      them belong to the model, which is out of scope).
  M4  HCA rows and window rows are always attended, whatever Level 2 selects (BJ north_star).

Functions: l2_native_scores, l2_resident_entries (M1), l2_topk_entries (Eq.6, M2),
l2_gather_kv / l2_decode_attention.  Pins: tests/test_l2_oracle_pins.py.
"""
from __future__ import annotations

from typing import Sequence, Tuple

import numpy as np

from .lsa_oracle import attention, widen


def l2_native_scores(q_idx: np.ndarray, w_idx: np.ndarray, index_k: np.ndarray) -> np.ndarray:
    """Score_native(i, s) for every row s of index_k.  q_idx [n_h][c_I], w_idx [n_h], index_k [n][c_I] -> [n]."""
    K = widen(index_k)
    q = widen(q_idx)
    w = np.asarray(w_idx, dtype=np.float64)
    match = K @ q.T                               # [n][n_h]: q_{i,h} . K_s
    return np.maximum(match, 0.0) @ w             # sum_h w_{i,h} ReLU(.)


def l2_resident_entries(table_chunks: Sequence[int], n_csa: int, C: int) -> np.ndarray:
    """M1: entry ids s = c*C + r of the valid rows of the chunks in the current table, ascending."""
    ids = []
    for c in sorted(int(c) for c in table_chunks):
        ids.extend(range(c * C, min(n_csa, (c + 1) * C)))
    return np.asarray(ids, dtype=np.int64)


def l2_topk_entries(scores: np.ndarray, entry_ids: np.ndarray, k2: int) -> np.ndarray:
    """Eq.(6), M2.  scores[j] belongs to entry_ids[j].  Returns the chosen entry ids in (score desc, id asc) order."""
    order = sorted(range(len(entry_ids)), key=lambda j: (-float(scores[j]), int(entry_ids[j])))
    return np.asarray([int(entry_ids[j]) for j in order[:max(0, k2)]], dtype=np.int64)


def l2_select(q_idx: np.ndarray, w_idx: np.ndarray, index_k: np.ndarray, table_chunks: Sequence[int], n_csa: int, C: int,
              k2: int) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """One sequence, one decode step: (selected entry ids, resident entry ids, their native scores)."""
    ids = l2_resident_entries(table_chunks, n_csa, C)
    K = np.asarray(index_k)[ids] if len(ids) else np.zeros((0, np.asarray(index_k).shape[1]), dtype=np.asarray(index_k).dtype)
    sc = l2_native_scores(q_idx, w_idx, K)
    return l2_topk_entries(sc, ids, k2), ids, sc


def l2_gather_kv(oracle, b: int, sel_entries: Sequence[int]):
    """HCA rows (+) the selected entries' rows of their hot pages (+) window rows [0, w_len).
    `oracle` is an LsaOracle (pool state, HCA, window); entries are read from the page their chunk occupies."""
    C = oracle.C
    page_of = {c: p for c, p in oracle.pool.cur[b]}
    Ks, Vs = [widen(oracle.hca_k[b])], [widen(oracle.hca_v[b])]
    for s in sorted(int(s) for s in sel_entries):
        c, r = divmod(s, C)
        page = oracle.pool.hot[page_of[c]]
        Ks.append(widen(page[0, r:r + 1]))
        Vs.append(widen(page[1, r:r + 1]))
    Ks.append(widen(oracle.win_k[b][: oracle.w_len[b]]))
    Vs.append(widen(oracle.win_v[b][: oracle.w_len[b]]))
    return np.concatenate(Ks, axis=0), np.concatenate(Vs, axis=0)


def l2_decode_attention(oracle, q: np.ndarray, sel_entries: Sequence[Sequence[int]]):
    """q [B,H,D] stored dtype; sel_entries[b] = Level-2 selection of sequence b -> out [B,H,D], lse [B,H] (float64)."""
    out = np.zeros((oracle.B, oracle.H, oracle.D))
    lse = np.full((oracle.B, oracle.H), -np.inf)
    for b in range(oracle.B):
        K, V = l2_gather_kv(oracle, b, sel_entries[b])
        out[b], lse[b], _ = attention(widen(q[b]), K, V, oracle.sm_scale)
    return out, lse


def validate_l2_selection(gpu_sel: Sequence[int], entry_ids: np.ndarray, scores: np.ndarray, k2: int, rel: float = 1e-5):
    """GPU selection (entry ids, -1 padded) vs the oracle's scores: the SET must be the oracle's except for swaps
    among entries whose oracle score lies within `rel` (relative) of the k2-th score (BASELINE.json's rule for
    top-k).  Returns None or a message."""
    g = [int(s) for s in gpu_sel if int(s) >= 0]
    want = min(k2, len(entry_ids))
    if len(g) != want:
        return f"{len(g)} entries selected, expected {want}"
    if len(set(g)) != len(g):
        return "duplicate entry ids"
    sc = {int(e): float(s) for e, s in zip(entry_ids, scores)}
    if any(s not in sc for s in g):
        return "selected an entry that is not resident / not valid"
    if want == 0 or want == len(entry_ids):
        return None
    ranked = sorted(sc, key=lambda e: (-sc[e], e))
    cut = sc[ranked[want - 1]]
    band = rel * max(abs(cut), 1e-30)
    gs = set(g)
    for e in ranked:
        if sc[e] > cut + band and e not in gs:
            return f"entry {e} (score {sc[e]}) is above the cut-off {cut} but missing"
    for e in g:
        if sc[e] < cut - band:
            return f"entry {e} (score {sc[e]}) is below the cut-off {cut}"
    return None
