"""CPU oracle for the Lookahead Sparse Attention (LSA) decode hot path.

TEST INFRASTRUCTURE - NOT PRODUCT CODE.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s cpu_baseline / `--impl reference` legs may import this package.  It shares
no code with the CUDA path (`paper_2606_09079_b200/csrc`, `paper_2606_09079_b200/lsa.py`)
and never imports it; the only thing both sides read is the stored input arrays made by
`paper_2606_09079_b200/workloads.py`.

Plain, slow and meant to be checked against the paper by eye: every quantity is computed
in float64 from the STORED (fp32- or bf16-rounded) inputs with numpy; library primitives
used as steps are `@` (matmul), `np.lexsort` / `sorted`, `np.exp`, `np.log`.  No blocking,
fusion or reordering beyond the definitions below.

`P:n` = /root/reference/PAPER.md line n.  `BJ` = BASELINE.json north_star / configs.
`R#` = the numbered readings in DESIGN.md ("Readings of the paper").

Functions and the passages they follow
  O1 trigger_fires      P:59 "t (mod tau) = 0"; "first fires at decode step 0"
  O2 query_tower        P:61-65 Eq.(1)-(2) collapsed to one linear map + L2 norm, the
                        "standard dual-encoder" of P:124 as fixed by BJ north_star (R1)
  O3 chunk_scores       P:71-75 Eq.(4) in BJ's form: cosine of the query embedding with one
                        precomputed embedding per CSA chunk (R1, R3)
  O4 topk_select        P:77-79 Eq.(5) with the threshold replaced by BJ's per-sequence
                        top-k, K_max := k, order (score desc, chunk idx asc) (R2, R14)
  O5 ResidencyOracle    P:179, P:185 (CPU cold mirror / GPU reserve, page-granular recall),
                        P:187 (residency bitmap + remap), P:189 (visible at t+1) (R9-R13)
  O6 attention          P:85 (selected entries (+) sliding-window KV -> core MQA attention),
                        P:185/P:197 (HCA always resident), one softmax over the union (R5)
  O8 merge_partials     the (m, l, o) merge identity of split softmax (BJ "combine kernel")
  LsaOracle.step        the per-step order S0..S8 of DESIGN.md

Pins (tests/test_oracle_pins.py): see DESIGN.md "Oracle pins".  Real-indexer behaviour
(which chunks a TRAINED indexer picks on real text) has no pin: parity unpinned, out of
scope - the paper prints no worked numeric example for this path.
"""
from __future__ import annotations

import math
from typing import List, Optional, Sequence, Tuple

import numpy as np

EPS_NORM = 1e-12  # R16: zero-norm clamp


# ----------------------------------------------------------------------------------------
# storage -> float64 (exact widening; the oracle's own copy, deliberately not shared)
# ----------------------------------------------------------------------------------------
def widen(x: np.ndarray) -> np.ndarray:
    """float32 array or uint16 bfloat16 bit patterns -> float64, exactly."""
    if x.dtype == np.uint16:
        return (x.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)
    return np.asarray(x, dtype=np.float64)


# ----------------------------------------------------------------------------------------
# O1  trigger
# ----------------------------------------------------------------------------------------
def trigger_fires(step: int, tau: int) -> bool:
    return step % tau == 0


# ----------------------------------------------------------------------------------------
# O2  query tower                                                 P:61-65, BJ
# ----------------------------------------------------------------------------------------
def query_tower(W_q: np.ndarray, h: np.ndarray) -> np.ndarray:
    """z_e = sum_d W[e,d] h[d];  q_hat = z / max(||z||_2, 1e-12).   W_q [E,Dh], h [Dh]."""
    z = widen(W_q) @ widen(h)
    return z / max(math.sqrt(float(np.sum(z * z))), EPS_NORM)


# ----------------------------------------------------------------------------------------
# O3  chunk scores                                                P:71-75 (BJ form)
# ----------------------------------------------------------------------------------------
def chunk_scores(q_hat: np.ndarray, chunk_emb: np.ndarray) -> np.ndarray:
    """score_c = sum_e q_hat[e] * Emb[c,e]; Emb rows are NOT re-normalised (stored = truth)."""
    return widen(chunk_emb) @ q_hat


# ----------------------------------------------------------------------------------------
# O4  top-k                                                       P:77-79, BJ
# ----------------------------------------------------------------------------------------
def topk_select(scores: np.ndarray, k: int) -> Tuple[np.ndarray, np.ndarray]:
    """First k_eff = min(k, n) chunk ids ordered by (score desc, chunk idx asc).

    Returns (sel_idx[k] int32 padded with -1, sel_score[k] float64 padded with -inf)."""
    n = len(scores)
    idx = np.arange(n)
    order = np.lexsort((idx, -scores))        # last key is primary: -score asc, then idx asc
    k_eff = min(k, n)
    sel = np.full(k, -1, dtype=np.int32)
    val = np.full(k, -np.inf, dtype=np.float64)
    sel[:k_eff] = order[:k_eff]
    val[:k_eff] = scores[order[:k_eff]]
    return sel, val


# ----------------------------------------------------------------------------------------
# O6  attention                                                   P:85, BJ
# ----------------------------------------------------------------------------------------
def attention(q: np.ndarray, K: np.ndarray, V: np.ndarray, sm_scale: float):
    """q [H,D], K [N,D], V [N,D] (already float64) -> (out [H,D], lse [H], p [H,N]).

    s_j = sm_scale * q_h . K_j ;  m = max_j s_j ;  p_j = exp(s_j - m) / sum_i exp(s_i - m)
    o_h = sum_j p_j V_j ;  lse = m + log(sum_i exp(s_i - m)).   N = 0 -> out 0, lse -inf."""
    H, D = q.shape
    if K.shape[0] == 0:
        return np.zeros((H, D)), np.full(H, -np.inf), np.zeros((H, 0))
    s = sm_scale * (q @ K.T)
    m = s.max(axis=1, keepdims=True)
    e = np.exp(s - m)
    l = e.sum(axis=1, keepdims=True)
    p = e / l
    return p @ V, (m + np.log(l))[:, 0], p


# ----------------------------------------------------------------------------------------
# O8  split merge                                                 BJ "combine kernel"
# ----------------------------------------------------------------------------------------
def partial_attention(q, K, V, sm_scale):
    """Un-normalised partial of one key split: (m [H], l [H], o [H,D]) with o = sum e^{s-m} V."""
    s = sm_scale * (q @ K.T)
    m = s.max(axis=1)
    e = np.exp(s - m[:, None])
    return m, e.sum(axis=1), e @ V


def merge_partials(parts: Sequence[Tuple[np.ndarray, np.ndarray, np.ndarray]]):
    """m* = max m_i ; l* = sum l_i e^{m_i-m*} ; out = sum o_i e^{m_i-m*} / l* ; lse = m* + log l*."""
    m_star = np.max(np.stack([p[0] for p in parts]), axis=0)
    l_star = sum(p[1] * np.exp(p[0] - m_star) for p in parts)
    o_star = sum(p[2] * np.exp(p[0] - m_star)[:, None] for p in parts)
    return o_star / l_star[:, None], m_star + np.log(l_star)


# ----------------------------------------------------------------------------------------
# O5  residency: shared paged hot pool with deterministic LRU      P:179-189, BJ cfg 4
# ----------------------------------------------------------------------------------------
class PoolExhausted(RuntimeError):
    pass


class ResidencyOracle:
    """State: owner[p] in {None,(b,c)}, page_of[b][c], last_used[p], tick; per sequence the
    current table `cur`, the staged table `nxt` (pending) and `visible_at`.

    fetch(b, selection): drop b's own pending table; tick += 1; S_up = selection sorted by
    chunk id.  pinned = pages of cur[b'] for all b' and of pending nxt[b'] (b' != b), plus
    pages touched in this call.  Pass 1: resident chunks of S_up are hits (last_used = tick,
    pinned).  Pass 2: the others, in ascending chunk id, each take the unpinned page
    minimising (last_used, page index) - never-used pages have last_used = 0, so the
    lowest-numbered free page wins first (R12); the previous owner is evicted; bytes are
    copied from the cold pool.  nxt[b] = [(c, page)] in ascending c (R13)."""

    def __init__(self, n_seqs: int, n_chunks: Sequence[int], hot_pages: int,
                 cold: Optional[Sequence[np.ndarray]] = None, cold_page_nbytes: Optional[int] = None):
        """cold_page_nbytes: bytes one page occupies in the cold pool when that differs from the hot image (FP8 cold pages,
        DESIGN R34: `cold` then holds the DEQUANTISED page images, which is what a recall writes into the hot pool)."""
        self.cold_page_nbytes = cold_page_nbytes
        self.P = int(hot_pages)
        self.owner: List[Optional[Tuple[int, int]]] = [None] * self.P
        self.last_used = [0] * self.P
        self.page_of = [[-1] * int(n) for n in n_chunks]
        self.tick = 0
        self.cur: List[List[Tuple[int, int]]] = [[] for _ in range(n_seqs)]
        self.nxt: List[Optional[List[Tuple[int, int]]]] = [None] * n_seqs
        self.visible_at = [0] * n_seqs
        self.cold = cold
        self.hot = None
        if cold is not None:
            self.hot = np.zeros((self.P,) + cold[0].shape[1:], dtype=cold[0].dtype)
        # counters (lsa_get_stats)
        self.hits = self.misses = self.evictions = self.triggers = 0
        self.bytes_fetched = 0

    def _pinned(self, b: int) -> set:
        pins = set()
        for bb in range(len(self.cur)):
            pins.update(p for _, p in self.cur[bb])
            if bb != b and self.nxt[bb] is not None:
                pins.update(p for _, p in self.nxt[bb])
        return pins

    def fetch(self, b: int, selection: Sequence[int], step_b: int, recall_lag: int):
        """Returns the fetch list [(chunk, page)] of this call (misses, ascending chunk)."""
        sel_up = sorted(int(c) for c in selection if c >= 0)
        self.nxt[b] = None                      # a new selection supersedes an unswapped one
        self.tick += 1
        self.triggers += 1
        pinned = self._pinned(b)
        for c in sel_up:                        # pass 1: hits
            p = self.page_of[b][c]
            if p >= 0:
                self.hits += 1
                self.last_used[p] = self.tick
                pinned.add(p)
        fetch_list = []
        for c in sel_up:                        # pass 2: misses, ascending chunk id
            if self.page_of[b][c] >= 0:
                continue
            cand = [(self.last_used[p], p) for p in range(self.P) if p not in pinned]
            if not cand:
                raise PoolExhausted(f"no unpinned page for seq {b} chunk {c}")
            _, p = min(cand)
            if self.owner[p] is not None:
                ob, oc = self.owner[p]
                self.page_of[ob][oc] = -1
                self.evictions += 1
            self.owner[p] = (b, c)
            self.page_of[b][c] = p
            self.last_used[p] = self.tick
            pinned.add(p)
            self.misses += 1
            fetch_list.append((c, p))
            if self.hot is not None:
                self.hot[p] = self.cold[b][c]   # byte copy of one page
                self.bytes_fetched += self.cold_page_nbytes or self.cold[b][c].nbytes
        self.nxt[b] = [(c, self.page_of[b][c]) for c in sel_up]
        self.visible_at[b] = step_b + recall_lag
        return fetch_list

    def maybe_swap(self, b: int, step_b: int) -> bool:
        """the staged table becomes the attended one once step_b >= visible_at."""
        if self.nxt[b] is not None and step_b >= self.visible_at[b]:
            self.cur[b] = self.nxt[b]
            self.nxt[b] = None
            return True
        return False


# ----------------------------------------------------------------------------------------
# the whole path, step by step
# ----------------------------------------------------------------------------------------
class LsaOracle:
    """Holds the same inputs as lsa_init_pools and replays S0..S8 per step.

    Step order, for every sequence b with counter step_b:
      (a) if a staged table is due (step_b >= visible_at) it becomes current       [S6]
      (b) if step_b % tau == 0: query tower, scores, top-k, residency + fetch,
          visible_at = step_b + recall_lag                                        [S0-S5]
      (c) if recall_lag == 0 the table staged in (b) becomes current now           [S6]
      (d) k_new/v_new (if given) are written to the window ring slot w_head         [S7 input]
      (e) attention over HCA (+) pages of cur (+) window rows [0, w_len)            [S7/S8]
      (f) step_b += 1
    """

    def __init__(self, *, dtype: str, H: int, D: int, C: int, W: int, k: int, tau: int,
                 recall_lag: int, hot_pages: int, W_q: np.ndarray,
                 cold_csa: Sequence[np.ndarray], n_csa: Sequence[int],
                 chunk_emb: Sequence[np.ndarray], hca_k, hca_v, win_k, win_v,
                 w_len: Sequence[int], w_head: Sequence[int], step0: Sequence[int],
                 sm_scale: float = 0.0, cold_page_nbytes: Optional[int] = None):
        self.dtype, self.H, self.D, self.C, self.W = dtype, H, D, C, W
        self.k, self.tau, self.recall_lag = k, tau, recall_lag
        self.sm_scale = sm_scale if sm_scale > 0 else 1.0 / math.sqrt(D)
        self.B = len(cold_csa)
        self.W_q = W_q
        self.cold = list(cold_csa)
        self.n_csa = [int(x) for x in n_csa]
        self.n_chunks = [-(-n // C) for n in self.n_csa]
        self.chunk_emb = list(chunk_emb)
        self.hca_k, self.hca_v = list(hca_k), list(hca_v)
        self.win_k = [x.copy() for x in win_k]
        self.win_v = [x.copy() for x in win_v]
        self.w_len, self.w_head = list(w_len), list(w_head)
        self.step = [int(s) for s in step0]
        self.pool = ResidencyOracle(self.B, self.n_chunks, hot_pages, self.cold, cold_page_nbytes)

    # -- S1-S3 ---------------------------------------------------------------------------
    def scores(self, b: int, h_b: np.ndarray) -> np.ndarray:
        return chunk_scores(query_tower(self.W_q, h_b), self.chunk_emb[b])

    def index_select(self, b: int, h_b: np.ndarray):
        return topk_select(self.scores(b, h_b), self.k)

    # -- S7 inputs -----------------------------------------------------------------------
    def valid_rows(self, b: int, c: int) -> int:
        return min(self.C, self.n_csa[b] - c * self.C)

    def gather_kv(self, b: int, table: Optional[Sequence[Tuple[int, int]]] = None):
        """Concatenate HCA rows, rows [0, valid(c)) of each page of the table, window rows."""
        table = self.pool.cur[b] if table is None else table
        Ks, Vs = [widen(self.hca_k[b])], [widen(self.hca_v[b])]
        for c, p in table:
            v = self.valid_rows(b, c)
            page = self.pool.hot[p]
            Ks.append(widen(page[0, :v]))
            Vs.append(widen(page[1, :v]))
        Ks.append(widen(self.win_k[b][: self.w_len[b]]))
        Vs.append(widen(self.win_v[b][: self.w_len[b]]))
        return np.concatenate(Ks, axis=0), np.concatenate(Vs, axis=0)

    def decode_attention(self, q: np.ndarray, seqs: Optional[Sequence[int]] = None):
        """q [B,H,D] stored dtype -> out [B,H,D] float64, lse [B,H] float64 (cur tables only)."""
        out = np.zeros((self.B, self.H, self.D))
        lse = np.full((self.B, self.H), -np.inf)
        for b in (range(self.B) if seqs is None else seqs):
            K, V = self.gather_kv(b)
            out[b], lse[b], _ = attention(widen(q[b]), K, V, self.sm_scale)
        return out, lse

    def append_window(self, b: int, k_new_b: np.ndarray, v_new_b: np.ndarray):
        self.win_k[b][self.w_head[b]] = k_new_b
        self.win_v[b][self.w_head[b]] = v_new_b
        self.w_head[b] = (self.w_head[b] + 1) % self.W
        self.w_len[b] = min(self.W, self.w_len[b] + 1)

    # -- the step ------------------------------------------------------------------------
    def step_begin(self, h: Optional[np.ndarray], forced_selection=None):
        """(a)-(c): swaps and trigger work.  Returns {b: (sel_idx, sel_score, fetch_list)}.

        forced_selection: optional {b: chunk ids} used INSTEAD of the oracle's own top-k when
        calling the residency model - the lock-step mode of the tolerance cascade
        (DESIGN.md): the caller first validates the GPU selection against O4, then feeds it
        here so page tables stay bit-comparable."""
        fired = {}
        for b in range(self.B):
            self.pool.maybe_swap(b, self.step[b])                        # (a)
        for b in range(self.B):                                          # (b) ascending b
            if trigger_fires(self.step[b], self.tau):
                sel, val = self.index_select(b, h[b])
                use = sel if forced_selection is None else np.asarray(forced_selection[b])
                fl = self.pool.fetch(b, use, self.step[b], self.recall_lag)
                fired[b] = (sel, val, fl)
        if self.recall_lag == 0:                                         # (c)
            for b in fired:
                self.pool.maybe_swap(b, self.step[b])
        return fired

    def step_end(self, q, k_new=None, v_new=None, attend: bool = True, seqs=None):
        """(d)-(f).  attend=False skips the (expensive) attention evaluation."""
        if k_new is not None:
            for b in range(self.B):
                self.append_window(b, k_new[b], v_new[b])                # (d)
        res = self.decode_attention(q, seqs) if attend else None         # (e)
        for b in range(self.B):
            self.step[b] += 1                                            # (f)
        return res

    def run_step(self, q, h, k_new=None, v_new=None, attend: bool = True, forced_selection=None):
        fired = self.step_begin(h, forced_selection)
        res = self.step_end(q, k_new, v_new, attend)
        return fired, res


def validate_selection(gpu_sel: np.ndarray, oracle_scores: np.ndarray, k: int,
                       rel_band: float = 1e-5) -> Optional[str]:
    """Check a GPU selection against O4 under BJ's tolerance.  None = OK, else a message.

    Outside the band {c : |score_c - score_(k)| <= rel_band*|score_(k)|} the selected SET must
    equal the oracle's; inside it any choice of the right cardinality passes, except that among
    bit-identical oracle scores the lower chunk id must win.  Order: non-increasing oracle score
    up to the band, and ascending chunk id among bit-identical scores."""
    n = len(oracle_scores)
    k_eff = min(k, n)
    g = [int(c) for c in gpu_sel[:k_eff]]
    if any(c < 0 or c >= n for c in g):
        return f"out-of-range chunk id in {g}"
    if len(set(g)) != k_eff:
        return "duplicate chunk ids"
    if any(int(c) != -1 for c in gpu_sel[k_eff:]):
        return "padding slots must be -1"
    o_sel, _ = topk_select(oracle_scores, k)
    kth = float(oracle_scores[o_sel[k_eff - 1]])
    band = rel_band * abs(kth)
    in_band = lambda c: abs(float(oracle_scores[c]) - kth) <= band
    must = {int(c) for c in range(n) if oracle_scores[c] > kth and not in_band(c)}
    if not must.issubset(g):
        return f"missing strictly-better chunks {sorted(must - set(g))}"
    for c in g:
        if c not in must and not in_band(c):
            return f"chunk {c} (score {oracle_scores[c]}) is below the k-th score band ({kth})"
    # exact ties: a selected chunk may not have an unselected bit-identical twin with a lower id
    gs = set(g)
    for c in g:
        twins = np.nonzero(oracle_scores == oracle_scores[c])[0]
        for t in twins:
            if int(t) < c and int(t) not in gs:
                return f"tie-break violated: chunk {c} selected but equal-score chunk {int(t)} is not"
    # order
    for a, bb in zip(g[:-1], g[1:]):
        sa, sb = float(oracle_scores[a]), float(oracle_scores[bb])
        if sa == sb:
            if a > bb:
                return f"equal scores out of index order: {a} before {bb}"
        elif sa < sb and (sb - sa) > rel_band * max(abs(sa), abs(sb)):
            return f"scores out of order: {a}({sa}) before {bb}({sb})"
    return None
