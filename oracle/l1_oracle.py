"""CPU oracle for the paper-exact Level-1 Memory Indexer.

TEST INFRASTRUCTURE - NOT PRODUCT CODE (same rules as oracle/lsa_oracle.py: only tests/, smoke() and
bench.py's cpu_baseline legs may import it; it shares no code with the CUDA path).

Plain numpy, float64 from the STORED (bf16- / fp32-rounded) inputs, in the paper's order and notation
(`P:n` = /root/reference/PAPER.md line n):

  Eq.(1)  c_t^Q = h_t . W^DQ                      W^DQ  in R^{d x d_c}
  Eq.(2)  q_t   = c_t^Q . W^IUQ                   W^IUQ in R^{d_c x (c^I n_h)}, n_h heads
  Eq.(3)  w_t   = h_t . W^w                       W^w   in R^{d x n_h}
  Eq.(4)  I_{t,s} = sigmoid( sum_h w_{t,h} ReLU( q_{t,h} . K_s^IComp ) )   per entry s
  Eq.(5)  recall { s : I_{t,s} >= 0.5 }, bounded by K_max
  Eq.(13) OR-union over the indexer layers

Readings:
  L1  storage: every weight is stored TRANSPOSED, [out][in] row-major (W_dq [d_c][d], W_iuq [n_h*c_I][d_c],
      W_w [n_h][d]); head h owns rows [h*c_I, (h+1)*c_I) of W_iuq.  Pure layout, no arithmetic change.
  L2  recall is page granular ("recall is in pages"): chunk c is recalled iff ANY of its valid
      entries meets the threshold in ANY layer; its score is the maximum I over its entries and layers.
  L3  K_max: if more than K_max chunks qualify, the K_max with the highest score are kept, ties by
      ascending chunk id (the paper gives no rule; same tie-break as BASELINE.json's top-k).
  L4  Eq.(4)-(5) taken literally: an entry whose gated sum is exactly 0 has I = 0.5 and IS recalled.
  L5  s ranges over all valid compressed entries of the sequence (the paper's s < floor(t/m)); the
      compressed history is static during a run (DESIGN R8).

Functions: l1_query (Eq.1-3), l1_entry_scores (Eq.4), l1_chunk_scores (L2), l1_select (Eq.5, 13, L3).
Pins: tests/test_l1_oracle_pins.py.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np


def _widen(x: np.ndarray) -> np.ndarray:
    """float32 array or uint16 bfloat16 bit patterns -> float64, exactly (own copy, not shared)."""
    if x.dtype == np.uint16:
        return (x.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)
    return np.asarray(x, dtype=np.float64)


def sigmoid(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):                 # exp(+large) -> inf -> 1/(1+inf) = 0, the right limit
        return 1.0 / (1.0 + np.exp(-np.asarray(x, dtype=np.float64)))


def l1_query(h: np.ndarray, W_dq: np.ndarray, W_iuq: np.ndarray, W_w: np.ndarray, n_h: int) -> Tuple[np.ndarray, np.ndarray]:
    """Eq.(1)-(3).  h [d]; W_dq [d_c][d]; W_iuq [n_h*c_I][d_c]; W_w [n_h][d]  ->  q [n_h][c_I], w [n_h]."""
    h = _widen(h)
    c_q = _widen(W_dq) @ h                       # Eq.(1)
    q = _widen(W_iuq) @ c_q                      # Eq.(2)
    w = _widen(W_w) @ h                          # Eq.(3)
    return q.reshape(n_h, -1), w


def l1_entry_scores(q: np.ndarray, w: np.ndarray, index_k: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """Eq.(4).  q [n_h][c_I], w [n_h], index_k [n_entries][c_I]  ->  (I [n_entries], pre-activation [n_entries])."""
    K = _widen(index_k)
    match = K @ q.T                              # [n_entries][n_h]:  q_{t,h} . K_s
    pre = np.maximum(match, 0.0) @ w             # sum_h w_h ReLU(.)
    return sigmoid(pre), pre


def l1_chunk_scores(I_layers: Sequence[np.ndarray], C: int) -> np.ndarray:
    """L2: score of chunk c = max over layers and over its valid entries of I."""
    n = len(I_layers[0])
    n_chunks = (n + C - 1) // C
    best = np.max(np.stack([np.asarray(x, dtype=np.float64) for x in I_layers]), axis=0)
    out = np.full(n_chunks, -np.inf)
    for c in range(n_chunks):
        out[c] = best[c * C:min(n, (c + 1) * C)].max()
    return out


def l1_select(chunk_score: np.ndarray, k_max: int, threshold: float = 0.5) -> Tuple[np.ndarray, np.ndarray]:
    """Eq.(5), (13), L3: chunks with score >= threshold, at most k_max of them by (score desc, idx asc).
    Returns (sel_idx[k_max] int32 padded with -1, sel_score[k_max] padded with -inf)."""
    cand = [c for c in range(len(chunk_score)) if chunk_score[c] >= threshold]
    cand.sort(key=lambda c: (-chunk_score[c], c))
    cand = cand[:k_max]
    sel = np.full(k_max, -1, dtype=np.int32)
    val = np.full(k_max, -np.inf)
    sel[:len(cand)] = cand
    val[:len(cand)] = [chunk_score[c] for c in cand]
    return sel, val


def l1_index_select(h: np.ndarray, layers: Sequence[dict], index_k: Sequence[np.ndarray], n_h: int, C: int, k_max: int,
                    threshold: float = 0.5):
    """Eq.(1)-(5), (13) for one sequence.  layers[l] = dict(W_dq, W_iuq, W_w); index_k[l] [n_entries][c_I].
    Returns (sel_idx, sel_score, chunk_score, per-layer pre-activations)."""
    I_layers, pre_layers = [], []
    for lay, K in zip(layers, index_k):
        q, w = l1_query(h, lay["W_dq"], lay["W_iuq"], lay["W_w"], n_h)
        I, pre = l1_entry_scores(q, w, K)
        I_layers.append(I)
        pre_layers.append(pre)
    cs = l1_chunk_scores(I_layers, C)
    sel, val = l1_select(cs, k_max, threshold)
    return sel, val, cs, pre_layers


def validate_l1_selection(gpu_sel: np.ndarray, chunk_score: np.ndarray, k_max: int, threshold: float, band: float):
    """GPU selection vs the oracle under a tolerance band (the GPU scores entries on bf16 tensor cores with a
    bf16-rounded query).  Chunks whose oracle score is within `band` of the threshold may go either way;
    outside it membership must match, except that when more than k_max qualify the cut-off score gets the
    same band.  Returns None or a message."""
    g = [int(c) for c in gpu_sel if int(c) >= 0]
    n_valid = len(g)
    if any(int(c) != -1 for c in gpu_sel[n_valid:]):
        return "valid ids must come first, then -1 padding"
    if len(set(g)) != len(g) or any(c >= len(chunk_score) for c in g):
        return "duplicate or out-of-range chunk ids"
    sure = [c for c in range(len(chunk_score)) if chunk_score[c] >= threshold + band]
    maybe = [c for c in range(len(chunk_score)) if abs(chunk_score[c] - threshold) < band]
    for c in g:
        if c not in sure and c not in maybe:
            return f"chunk {c} selected with oracle score {chunk_score[c]} < threshold {threshold}"
    if len(sure) + len(maybe) <= k_max:
        missing = [c for c in sure if c not in g]
        return f"qualifying chunks not selected: {missing}" if missing else None
    # capped: every chunk clearly above the cut-off must be in, nothing clearly below it
    ranked = sorted(sure + maybe, key=lambda c: (-chunk_score[c], c))
    cut = chunk_score[ranked[k_max - 1]]
    for c in ranked:
        if chunk_score[c] > cut + band and c not in g and chunk_score[c] >= threshold + band:
            return f"chunk {c} (score {chunk_score[c]}) is above the cut-off {cut} but missing"
    for c in g:
        if chunk_score[c] < cut - band:
            return f"chunk {c} (score {chunk_score[c]}) is below the cut-off {cut}"
    if len(g) > k_max:
        return "more than k_max chunks selected"
    if len(sure) >= k_max and len(g) != k_max:
        return f"{len(sure)} chunks clearly qualify but only {len(g)} of k_max = {k_max} were selected"
    return None
