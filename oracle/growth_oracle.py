"""CPU oracle for NEXT-4 (second half): the compressed history grows while decoding.

TEST INFRASTRUCTURE - NOT PRODUCT CODE (same rules as oracle/lsa_oracle.py: only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs import it; it shares no
code with the CUDA path).

What the paper states (P:n = /root/reference/PAPER.md line n):
  P:185  "The GPU resident set thus comprises four always-resident tiers - HCA layers (128:1 compression), the
         CSA chunks corresponding to the last 8K tokens of the original prompt (sliding window), all actively
         decoded tokens' CSA chunks, and the index-K [...] - plus the dynamically recalled CSA subset
         C_t^MemComp.  Everything else lives in the CPU cold mirror."
  P:179  the full KV is streamed into the D-side pinned host memory (VRAM -> DRAM), Fig. 4.
The paper does not say how an entry produced during decode enters that structure; the readings built
here (R29-R33):
  R29  the caller hands over already-compressed entries (one CSA entry every 4 tokens, one HCA entry every 128;
       the compressor itself needs the model) BEFORE the step that first attends them.
  R30  the chunk being filled (the "tail" chunk, id n_csa // C) is always resident and always attended with
       its valid rows: it is tier 3 of P:185.  It is NOT a candidate of the indexer (it has no embedding yet),
       so candidates are the FULL chunks only: n_chunks = n_csa // C.
  R31  when an entry completes a chunk, the chunk gets its embedding row, is mirrored to the cold pool
       (P:179 direction) and becomes a candidate from the next trigger on.  It stays attended through the
       tier until a table becomes current whose trigger already saw it as a candidate - from then on it is
       attended if and only if the indexer recalls it, like any chunk of the prompt (bounded HBM: the
       decode tier holds at most two chunks per sequence).
  R32  the tier lives in two reserved pages per sequence at the END of the hot pool, outside the LRU
       economy: page(b, c) = P_lru + 2 b + (c mod 2), P_lru = hot_pages - 2 B.  Tier entries follow the
       recalled entries in the page table (their chunk ids are larger than any candidate's: the table stays
       ascending, R13).
  R33  two of the k table slots are the tier's: at most k - 2 chunks are recalled (k_sel = k - 2).

O9 functions
  GrowingLsaOracle.append_compressed   R29-R31, one entry at a time
  GrowingLsaOracle.tier / table        R30-R32 written as a membership rule, not as table edits:
       tier(b) = { c : ncand_cur[b] <= c < ceil(n_csa / C) }, where ncand_cur[b] is the number of candidates
       seen by the trigger whose table is current (the initial number of full chunks before any swap).

Pins (tests/test_growth_oracle_pins.py): every attended set equals dense attention over the full grown
history when everything is recalled, and equals a run INITIALISED with the longer history; a hand-traced
tier schedule (tests/golden/growth_hand_case.json); invariants (each entry attended at most once, the tail
always attended, export bytes = appended rows, at most two tier chunks); without appends the class is the
static oracle with k - 2 and P - 2B.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import numpy as np

from .lsa_oracle import LsaOracle, ResidencyOracle, chunk_scores, query_tower, topk_select, trigger_fires, widen

TIER_SLOTS = 2          # R32 / R33


class TierOverflow(RuntimeError):
    """A third chunk would enter the decode tier before the oldest one has graduated (R31)."""


class GrowingLsaOracle(LsaOracle):
    """LsaOracle whose arrays have CAPACITY sizes: cold_csa[b] holds cap_chunks(b) pages, chunk_emb[b] cap_chunks(b)
    rows, hca_k / hca_v[b] cap_hca(b) rows; n_csa / n_hca give the rows in use."""

    def __init__(self, *, n_hca: Sequence[int], hot_pages: int, **kw):
        B = len(kw["cold_csa"])
        self.P_total = int(hot_pages)
        self.P_lru = self.P_total - TIER_SLOTS * B                     # R32
        super().__init__(hot_pages=self.P_lru, **kw)
        C = self.C
        self.n_hca = [int(x) for x in n_hca]
        self.cap_chunks = [int(x.shape[0]) for x in self.cold]
        self.n_chunks = [n // C for n in self.n_csa]                   # R30: candidates = full chunks
        self.k_sel = self.k - TIER_SLOTS                               # R33
        self.pool = ResidencyOracle(B, self.cap_chunks, self.P_lru, self.cold)
        hot = np.zeros((self.P_total,) + self.cold[0].shape[1:], dtype=self.cold[0].dtype)
        self.pool.hot = hot                                            # pages [P_lru, P_total) are the tier's
        self.ncand_cur = list(self.n_chunks)                           # candidates seen by the current table's trigger
        self.ncand_nxt = list(self.n_chunks)
        self.exported = 0
        for b in range(B):                                             # a partial last chunk of the prompt is the first tail
            if self.n_csa[b] % C:
                c = self.n_csa[b] // C
                hot[self.tier_page(b, c)] = self.cold[b][c]

    # -- R32 -----------------------------------------------------------------------------
    def tier_page(self, b: int, c: int) -> int:
        return self.P_lru + TIER_SLOTS * b + (c % TIER_SLOTS)

    def tier(self, b: int, ncand: Optional[int] = None) -> List[int]:
        """Chunks attended through the decode tier (R30/R31): started, and not yet seen as a candidate by the
        trigger of the table in question."""
        lo = self.ncand_cur[b] if ncand is None else ncand
        return list(range(lo, -(-self.n_csa[b] // self.C)))

    def table(self, b: int, which: int = 0) -> Optional[List[Tuple[int, int]]]:
        """which = 0: the attended table; 1: the staged one (None if nothing is pending)."""
        if which == 0:
            return list(self.pool.cur[b]) + [(c, self.tier_page(b, c)) for c in self.tier(b)]
        if self.pool.nxt[b] is None:
            return None
        return list(self.pool.nxt[b]) + [(c, self.tier_page(b, c)) for c in self.tier(b, self.ncand_nxt[b])]

    # -- R29-R31 ---------------------------------------------------------------------------
    def append_compressed(self, b: int, csa_k=None, csa_v=None, hca_k=None, hca_v=None, emb_row=None) -> bool:
        """Hand over one HCA entry and / or one CSA entry of sequence b.  Returns True if the CSA entry completed a chunk."""
        if hca_k is not None:
            if self.n_hca[b] >= self.hca_k[b].shape[0]:
                raise ValueError("HCA capacity exceeded")
            self.hca_k[b][self.n_hca[b]] = hca_k
            self.hca_v[b][self.n_hca[b]] = hca_v
            self.n_hca[b] += 1
        if csa_k is None:
            return False
        n, C = self.n_csa[b], self.C
        c, i = divmod(n, C)
        if c >= self.cap_chunks[b]:
            raise ValueError("CSA capacity exceeded")
        if i == 0 and len(self.tier(b)) >= TIER_SLOTS:
            raise TierOverflow(f"seq {b}: chunk {c} would be the third tier chunk")
        p = self.tier_page(b, c)
        self.pool.hot[p][0, i] = csa_k
        self.pool.hot[p][1, i] = csa_v
        self.n_csa[b] = n + 1
        if i != C - 1:
            return False
        if emb_row is None:
            raise ValueError("the entry completes a chunk: its embedding row is required")
        self.chunk_emb[b][c] = emb_row                                 # R31
        self.cold[b][c] = self.pool.hot[p]                             # export: byte copy of the page
        self.n_chunks[b] = c + 1
        self.exported += 1
        return True

    # -- S1-S3 over the candidates ------------------------------------------------------------
    def scores(self, b: int, h_b: np.ndarray) -> np.ndarray:
        return chunk_scores(query_tower(self.W_q, h_b), self.chunk_emb[b][: self.n_chunks[b]])

    def index_select(self, b: int, h_b: np.ndarray):
        sel, val = topk_select(self.scores(b, h_b), self.k_sel)
        pad = self.k - self.k_sel                                      # same [k] layout as the static path
        return (np.concatenate([sel, np.full(pad, -1, dtype=sel.dtype)]),
                np.concatenate([val, np.full(pad, -np.inf)]))

    # -- S7 inputs ---------------------------------------------------------------------------
    def gather_kv(self, b: int, table=None):
        table = self.table(b) if table is None else table
        Ks, Vs = [widen(self.hca_k[b][: self.n_hca[b]])], [widen(self.hca_v[b][: self.n_hca[b]])]
        for c, p in table:
            v = self.valid_rows(b, c)
            Ks.append(widen(self.pool.hot[p][0, :v]))
            Vs.append(widen(self.pool.hot[p][1, :v]))
        Ks.append(widen(self.win_k[b][: self.w_len[b]]))
        Vs.append(widen(self.win_v[b][: self.w_len[b]]))
        return np.concatenate(Ks, axis=0), np.concatenate(Vs, axis=0)

    # -- (a)-(c) with the candidate counts the tier rule needs -----------------------------------
    def step_begin(self, h, forced_selection=None):
        fired = {}
        for b in range(self.B):
            if self.pool.maybe_swap(b, self.step[b]):                    # (a)
                self.ncand_cur[b] = self.ncand_nxt[b]
        for b in range(self.B):                                          # (b) ascending b
            if trigger_fires(self.step[b], self.tau):
                sel, val = self.index_select(b, h[b])
                use = sel if forced_selection is None else np.asarray(forced_selection[b])
                fl = self.pool.fetch(b, use, self.step[b], self.recall_lag)
                self.ncand_nxt[b] = self.n_chunks[b]
                fired[b] = (sel, val, fl)
        if self.recall_lag == 0:                                         # (c)
            for b in fired:
                if self.pool.maybe_swap(b, self.step[b]):
                    self.ncand_cur[b] = self.ncand_nxt[b]
        return fired
