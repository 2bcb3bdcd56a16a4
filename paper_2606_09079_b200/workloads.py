"""Seeded synthetic LSA workloads (inputs only - none of the method's arithmetic).

This module is the ONE piece shared by the CUDA path (tests, bench.py) and the CPU
oracle (oracle/): it produces the stored, already-rounded input arrays that both sides
read.  It never scores, selects, allocates pages or attends.  It depends on numpy and
torch-CPU only and must stay importable without the CUDA extension.

Shapes / distributions follow BASELINE.json `configs` (numbered 1..5 here) and
SURVEY.md 8(d); the recipe is restated in DESIGN.md "Input recipe".  They stand in for
the paper's long-context workloads (Table 1 context lengths 46K-512K, Fig. 1
1M-token projection) - only the context-length range and the ~10 % recall ratio are
taken from the paper, no item of any benchmark suite.

Array conventions
-----------------
* dtype "f32": numpy float32 arrays.
* dtype "bf16": numpy uint16 arrays holding bfloat16 bit patterns (numpy has no bf16).
  `to_torch` / `as_f64` convert.  The stored bit patterns are the truth for both sides.
* cold_csa[b] : [n_chunks, 2, C, D]   (K block then V block per chunk = one page)
* chunk_emb[b]: [n_chunks, E]         hca_k/hca_v[b]: [n_hca, D]     win_k/win_v[b]: [W, D]
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional, Tuple

import numpy as np
import torch

BASE_SEED = 260609079 * 8  # seed = 260609079*8 + config_id


# --------------------------------------------------------------------------------------
# dtype helpers (storage only)
# --------------------------------------------------------------------------------------
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round float32 -> bfloat16 bit patterns (round-to-nearest-even), as uint16."""
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32))
    return t.to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16).copy()


def bf16_bits_to_f32(bits: np.ndarray) -> np.ndarray:
    return (bits.astype(np.uint32) << 16).view(np.float32)


def store(x: np.ndarray, dtype: str) -> np.ndarray:
    """Round a float array to the storage dtype of the config."""
    if dtype == "f32":
        return np.ascontiguousarray(x, dtype=np.float32)
    if dtype == "bf16":
        return f32_to_bf16_bits(np.asarray(x, dtype=np.float32))
    raise ValueError(dtype)


def as_f64(x: np.ndarray, dtype: str) -> np.ndarray:
    """Exact widening of a stored array to float64."""
    if dtype == "f32":
        return x.astype(np.float64)
    return bf16_bits_to_f32(x).astype(np.float64)


def to_torch(x: np.ndarray, dtype: str) -> torch.Tensor:
    """Stored numpy array -> torch CPU tensor of the matching dtype (shares memory)."""
    if dtype == "f32":
        return torch.from_numpy(x)
    return torch.from_numpy(x.view(np.int16)).view(torch.bfloat16)


def from_torch(t: torch.Tensor, dtype: str) -> np.ndarray:
    t = t.detach().cpu().contiguous()
    if dtype == "f32":
        return t.numpy()
    return t.view(torch.int16).numpy().view(np.uint16)


def elem_size(dtype: str) -> int:
    return 4 if dtype == "f32" else 2


# --------------------------------------------------------------------------------------
# configuration
# --------------------------------------------------------------------------------------
@dataclasses.dataclass
class LsaWorkloadConfig:
    name: str
    config_id: int
    dtype: str                 # "f32" | "bf16"
    B: int
    L: List[int]               # per-sequence context length in tokens
    H: int
    D: int
    C: int                     # CSA entries per chunk (= page rows)
    W: int                     # window capacity (raw tokens)
    Dh: int
    E: int
    k: int
    tau: int
    steps: int
    hot_pages: int
    recall_lag: int = 1
    csa_ratio: int = 4         # BASELINE.json cfg 1 "assumed 4:1"
    hca_ratio: int = 128       # PAPER.md l.31 "128:1"
    emb_mode: str = "beta"     # "needle0" (cfg1) | "beta" (cfg 2-4) | "uniform" (cfg 5)
    n_needles: int = 16
    needle_cos: float = 0.8
    needle_period: int = 4     # needles drift every this many triggers
    h_noise: float = 0.05
    stagger: bool = False      # cfg 4: per-sequence trigger phase
    tie_frac: float = 0.0      # cfg 5: fraction of triggers carrying planted ties
    q_gain: float = 1.0        # 1.0 = BASELINE recipe q ~ N(0,1)/sqrt(D)
    kv_base_chunks: int = 0    # >0: cold pools are tiled from this many random chunks
    seq_offset: int = 0        # this config holds sequences [seq_offset, seq_offset + B) of a batch of B_total
    B_total: int = 0           # 0 = B (not a shard); see shard_config()

    # ---- derived per sequence -------------------------------------------------------
    def n_hca(self, b: int) -> int:
        return self.L[b] // self.hca_ratio

    def n_csa(self, b: int) -> int:
        return self.L[b] // self.csa_ratio

    def n_chunks(self, b: int) -> int:
        return -(-self.n_csa(b) // self.C)

    def k_eff(self, b: int) -> int:
        return min(self.k, self.n_chunks(b))

    def step0(self, b: int) -> int:
        if not self.stagger:
            return 0
        # sequence b first fires at global step (b*tau//B) mod tau (b, B of the whole batch)
        return (self.tau - ((b + self.seq_offset) * self.tau // (self.B_total or self.B)) % self.tau) % self.tau

    @property
    def page_elems(self) -> int:
        return 2 * self.C * self.D

    @property
    def page_bytes(self) -> int:
        return self.page_elems * elem_size(self.dtype)

    @property
    def seed(self) -> int:
        return BASE_SEED + self.config_id

    def keys_attended(self, b: int, selected: bool = True) -> int:
        """N_b of SURVEY 8: HCA rows + selected chunks (full pages) + full window."""
        return self.n_hca(b) + (self.k_eff(b) * self.C if selected else 0) + min(self.W, self.L[b])

    def attn_bytes_per_step(self) -> int:
        """Algorithmic bytes of S7 per step, all sequences."""
        sz = elem_size(self.dtype)
        return sum(self.keys_attended(b) * 2 * self.D * sz + 2 * self.H * self.D * sz
                   for b in range(self.B))

    def attn_flops_per_step(self) -> int:
        return sum(4 * self.H * self.D * self.keys_attended(b) for b in range(self.B))


def _ragged_lengths(seed: int, B: int, lo: int, hi: int) -> List[int]:
    g = np.random.Generator(np.random.Philox(seed))
    u = g.uniform(math.log(lo), math.log(hi), size=B)
    return [int(math.floor(math.exp(x))) // 128 * 128 for x in u]


def make_config(config_id: int, **overrides) -> LsaWorkloadConfig:
    """The five BASELINE.json configs (1-based, file order)."""
    if config_id == 1:
        cfg = LsaWorkloadConfig(
            name="cfg1_tiny_f32_8k", config_id=1, dtype="f32", B=1, L=[8192], H=16, D=128,
            C=64, W=512, Dh=1024, E=256, k=4, tau=64, steps=128, hot_pages=8,
            emb_mode="needle0", n_needles=4, needle_cos=0.9, needle_period=10**9)
    elif config_id == 2:
        cfg = LsaWorkloadConfig(
            name="cfg2_bf16_128k", config_id=2, dtype="bf16", B=1, L=[131072], H=64, D=512,
            C=128, W=8192, Dh=4096, E=512, k=16, tau=64, steps=1024, hot_pages=64)
    elif config_id == 3:
        cfg = LsaWorkloadConfig(
            name="cfg3_bf16_1m", config_id=3, dtype="bf16", B=1, L=[1048576], H=64, D=512,
            C=128, W=8192, Dh=4096, E=512, k=64, tau=64, steps=2048,
            hot_pages=205)  # ceil(0.1 * 2048 chunks)
    elif config_id == 4:
        B = 32
        L = _ragged_lengths(BASE_SEED + 4, B, 65536, 1048576)
        cfg = LsaWorkloadConfig(
            name="cfg4_bf16_b32_ragged", config_id=4, dtype="bf16", B=B, L=L, H=64, D=512,
            C=128, W=8192, Dh=4096, E=512, k=32, tau=64, steps=512,
            hot_pages=16 * 10**9 // (2 * 128 * 512 * 2),  # 16e9 B -> 61035 pages
            stagger=True, kv_base_chunks=256)
    elif config_id == 5:
        B = 8
        cfg = LsaWorkloadConfig(
            name="cfg5_bf16_churn", config_id=5, dtype="bf16", B=B, L=[524288] * B, H=64,
            D=512, C=128, W=8192, Dh=4096, E=512, k=128, tau=16, steps=1024,
            hot_pages=2 * 128 * B,  # 2k pages per sequence
            emb_mode="uniform", n_needles=0, tie_frac=0.10, kv_base_chunks=256)
    else:
        raise ValueError(f"config_id must be 1..5, got {config_id}")
    return dataclasses.replace(cfg, **overrides) if overrides else cfg


def shard_config(cfg: LsaWorkloadConfig, lo: int, hi: int) -> LsaWorkloadConfig:
    """Sequences [lo, hi) of `cfg` as a config of their own (one rank's share when the batch is sharded by sequence):
    same per-sequence data and trigger phases as in the whole batch, the hot pool cut in proportion."""
    if not (0 <= lo < hi <= cfg.B):
        raise ValueError("bad shard")
    pages = max(2 * sum(min(cfg.k, -(-(cfg.L[b] // cfg.csa_ratio) // cfg.C)) for b in range(lo, hi)),
                cfg.hot_pages * (hi - lo) // cfg.B)
    return dataclasses.replace(cfg, B=hi - lo, L=list(cfg.L[lo:hi]), hot_pages=pages, seq_offset=cfg.seq_offset + lo,
                               B_total=cfg.B_total or cfg.B)


def make_small_config(dtype: str = "f32", **kw) -> LsaWorkloadConfig:
    """A scaled-down shape for CPU tests and fast parity cases (not a BASELINE config)."""
    base = dict(name="small", config_id=101, dtype=dtype, B=2, L=[4096, 2432], H=8, D=64, C=16,
                W=64, Dh=128, E=64, k=3, tau=4, steps=12, hot_pages=16, emb_mode="beta",
                n_needles=2, needle_cos=0.8, needle_period=2)
    base.update(kw)
    return LsaWorkloadConfig(**base)


# --------------------------------------------------------------------------------------
# generator
# --------------------------------------------------------------------------------------
def _rng(seed: int, *tags: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=np.random.SeedSequence([seed, *tags]).generate_state(2, np.uint64)))


def _randn_stored(g: np.random.Generator, shape, scale: float, dtype: str) -> np.ndarray:
    x = g.standard_normal(size=shape, dtype=np.float32)
    x *= np.float32(scale)
    return store(x, dtype)


def _unit_rows(x: np.ndarray) -> np.ndarray:
    return x / np.linalg.norm(x, axis=-1, keepdims=True)


class LsaWorkload:
    """All static inputs of one config plus per-step / per-trigger dynamic inputs."""

    def __init__(self, cfg: LsaWorkloadConfig, build_kv: bool = True):
        """build_kv=False skips every K/V array (indexer-only uses at full config sizes)."""
        self.cfg = cfg
        c = cfg
        dt = c.dtype
        s = c.seed
        self.W_q = _randn_stored(_rng(s, 1), (c.E, c.Dh), 1.0 / math.sqrt(c.Dh), dt)
        self.hca_k, self.hca_v, self.win_k, self.win_v = [], [], [], []
        self.cold_csa: List[np.ndarray] = []
        self.h0: List[np.ndarray] = []        # stored dtype [Dh]
        self.u: List[np.ndarray] = []         # float64 [E]: planted query direction
        self.base_cos: List[np.ndarray] = []  # float64 [n_chunks] (beta mode)
        self.base_emb: List[np.ndarray] = []  # stored [n_chunks, E]
        self._needle_cache: Dict[Tuple[int, int], np.ndarray] = {}
        inv_sqrt_d = 1.0 / math.sqrt(c.D)
        kv_base = None
        if c.kv_base_chunks > 0 and build_kv:
            kv_base = _randn_stored(_rng(s, 2), (c.kv_base_chunks, 2, c.C, c.D), inv_sqrt_d, dt)
        Wf = as_f64(self.W_q, dt)
        for b in range(c.B):
            nch = c.n_chunks(b)
            gb = b + c.seq_offset                   # index in the whole batch: a shard sees the same data
            if build_kv:
                self._build_kv(b, kv_base, inv_sqrt_d)

            # planted query direction u_b and an h0 with  W_q h0 = s*u  built by least squares
            # (np.linalg.lstsq min-norm solve - a construction, not the query tower itself).
            g = _rng(s, 20, gb)
            u = _unit_rows(g.standard_normal(c.E))
            gvec = g.standard_normal(c.Dh)
            zg = Wf @ gvec
            rhs = np.linalg.norm(zg) * u - zg
            corr = np.linalg.lstsq(Wf, rhs, rcond=None)[0]
            self.h0.append(store((gvec + corr).astype(np.float32), dt))
            self.u.append(u)

            ge = _rng(s, 21, gb)
            r = ge.standard_normal((nch, c.E))
            if c.emb_mode == "beta":
                cosv = ge.beta(2.0, 8.0, size=nch)
                self.base_cos.append(cosv)
                emb = self._plant(u, r, cosv)
            else:                                   # "needle0" / "uniform": random unit rows
                self.base_cos.append(np.zeros(nch))
                emb = _unit_rows(r)
            self.base_emb.append(store(emb.astype(np.float32), dt))

    def _build_kv(self, b: int, kv_base: Optional[np.ndarray], inv_sqrt_d: float) -> None:
        c, dt, s = self.cfg, self.cfg.dtype, self.cfg.seed
        nh, nch, ncsa = c.n_hca(b), c.n_chunks(b), c.n_csa(b)
        gb = b + c.seq_offset
        self.hca_k.append(_randn_stored(_rng(s, 10, gb), (nh, c.D), inv_sqrt_d, dt))
        self.hca_v.append(_randn_stored(_rng(s, 11, gb), (nh, c.D), inv_sqrt_d, dt))
        self.win_k.append(_randn_stored(_rng(s, 12, gb), (c.W, c.D), inv_sqrt_d, dt))
        self.win_v.append(_randn_stored(_rng(s, 13, gb), (c.W, c.D), inv_sqrt_d, dt))
        if kv_base is None:
            cold = _randn_stored(_rng(s, 14, gb), (nch, 2, c.C, c.D), inv_sqrt_d, dt)
        else:
            # tile the base block with a per-sequence stride so chunks differ per (b, c)
            idx = (np.arange(nch, dtype=np.int64) * 7 + 13 * gb) % c.kv_base_chunks
            cold = kv_base[idx].copy()
            # make every chunk unique in its first K element (cheap) so wrong copies are detectable
            tagv = store((((np.arange(nch) % 251) / 251.0 - 0.5) * inv_sqrt_d).astype(np.float32), dt)
            cold[:, 0, 0, 0] = tagv
        tail = nch * c.C - ncsa
        if tail:
            cold[nch - 1, :, c.C - tail:, :] = 0   # rows past n_csa: zero padding
        self.cold_csa.append(cold)

    # ---- embeddings -----------------------------------------------------------------
    @staticmethod
    def _plant(u: np.ndarray, r: np.ndarray, cosv: np.ndarray) -> np.ndarray:
        """rows = cos*u + sqrt(1-cos^2)*r_perp  with r_perp unit and orthogonal to u."""
        r_perp = r - (r @ u)[:, None] * u[None, :]
        r_perp = _unit_rows(r_perp)
        return cosv[:, None] * u[None, :] + np.sqrt(1.0 - cosv ** 2)[:, None] * r_perp

    def needle_ids(self, b: int, trigger_idx: int) -> np.ndarray:
        """Chunk ids carrying needles during trigger `trigger_idx` (drift every needle_period)."""
        c = self.cfg
        if c.n_needles == 0:
            return np.zeros(0, dtype=np.int64)
        epoch = trigger_idx // c.needle_period
        key = (b, epoch)
        if key not in self._needle_cache:
            g = _rng(c.seed, 30, b + c.seq_offset, epoch)
            n = min(c.n_needles, c.n_chunks(b))
            self._needle_cache[key] = np.sort(g.choice(c.n_chunks(b), size=n, replace=False))
        return self._needle_cache[key]

    def chunk_emb(self, b: int, trigger_idx: int) -> np.ndarray:
        """Embedding table [n_chunks, E] (stored dtype) in force at trigger `trigger_idx`."""
        c = self.cfg
        emb = self.base_emb[b].copy()
        ids = self.needle_ids(b, trigger_idx)
        if len(ids):
            g = _rng(c.seed, 31, b + c.seq_offset, trigger_idx // c.needle_period)
            r = g.standard_normal((len(ids), c.E))
            rows = self._plant(self.u[b], r, np.full(len(ids), c.needle_cos))
            emb[ids] = store(rows.astype(np.float32), c.dtype)
        return emb

    def emb_row_updates(self, b: int, trigger_idx: int) -> Optional[Tuple[np.ndarray, np.ndarray]]:
        """(row ids, new rows) to rewrite in place when the needle epoch changes, else None."""
        c = self.cfg
        if c.n_needles == 0 or trigger_idx == 0 or trigger_idx % c.needle_period != 0:
            return None
        old = self.needle_ids(b, trigger_idx - 1)
        new = self.needle_ids(b, trigger_idx)
        ids = np.union1d(old, new)
        return ids, self.chunk_emb(b, trigger_idx)[ids]

    # ---- per-step dynamic inputs ----------------------------------------------------
    def q(self, step: int) -> np.ndarray:
        c = self.cfg
        return _randn_stored(_rng(c.seed, 40, step), (c.B, c.H, c.D), c.q_gain / math.sqrt(c.D), c.dtype)

    def kv_new(self, step: int) -> Tuple[np.ndarray, np.ndarray]:
        c = self.cfg
        g = _rng(c.seed, 41, step)
        s = 1.0 / math.sqrt(c.D)
        return _randn_stored(g, (c.B, c.D), s, c.dtype), _randn_stored(g, (c.B, c.D), s, c.dtype)

    def h(self, step: int) -> np.ndarray:
        """Hidden states [B, Dh] at global step `step` (only consumed at trigger steps)."""
        c = self.cfg
        g = _rng(c.seed, 42, step)
        if c.emb_mode == "uniform":            # cfg 5: redrawn i.i.d. -> scores resampled
            return _randn_stored(g, (c.B, c.Dh), 1.0, c.dtype)
        out = np.empty((c.B, c.Dh), dtype=np.float32)
        for b in range(c.B):
            out[b] = as_f64(self.h0[b], c.dtype) + c.h_noise * g.standard_normal(c.Dh)
        return store(out, c.dtype)

    # ---- schedule helpers (integer bookkeeping of the harness, not the method) -------
    def seq_step(self, b: int, global_step: int) -> int:
        return self.cfg.step0(b) + global_step

    def fires(self, b: int, global_step: int) -> bool:
        return self.seq_step(b, global_step) % self.cfg.tau == 0

    def trigger_index(self, b: int, global_step: int) -> int:
        """Number of triggers of sequence b at global steps < global_step.

        At a firing step this is the 0-based index of that trigger (harness bookkeeping)."""
        c = self.cfg
        first = (-c.step0(b)) % c.tau          # first global step at which seq b fires
        if global_step <= first:
            return 0
        return (global_step - first - 1) // c.tau + 1

    def has_tie_trigger(self, b: int, trigger_idx: int) -> bool:
        c = self.cfg
        if c.tie_frac <= 0:
            return False
        g = _rng(c.seed, 50, b + c.seq_offset, trigger_idx)
        return bool(g.uniform() < c.tie_frac)

    def total_cold_bytes(self) -> int:
        return sum(x.nbytes for x in self.cold_csa)


def plant_boundary_ties(emb: np.ndarray, order: np.ndarray, k: int, dtype: str) -> np.ndarray:
    """Return a copy of `emb` with an exact tie and a near tie planted across the k-th rank.

    `order` is a ranking of chunk ids (best first) computed by the CALLER (tests use the
    oracle; bench.py uses any fixed permutation).  Row order[k] becomes a bit copy of row
    order[k-1] (exact tie across the boundary: the lower chunk id must win); row
    order[k+1] becomes that row with one low-magnitude coordinate moved by one ulp
    (score gap ~1e-6).  SURVEY 8(d) cfg 5, R14.
    """
    out = emb.copy()
    n = len(order)
    if k < 1 or k >= n:
        return out
    src = order[k - 1]
    out[order[k]] = out[src]
    if k + 1 < n:
        row = out[src].copy()
        mag = np.abs(as_f64(row, dtype))
        mag[mag == 0] = np.inf
        j = int(np.argmin(mag))
        if dtype == "bf16":
            row[j] = np.uint16(int(row[j]) ^ 1) if (int(row[j]) & 0x7FFF) != 0 else row[j]
        else:
            row[j] = np.nextafter(row[j], np.float32(0))
        out[order[k + 1]] = row
    return out


# --------------------------------------------------------------------------------------
# inputs of the paper-exact Level-1 indexer (Eq.(1)-(5), (13))
# --------------------------------------------------------------------------------------
class L1Inputs:
    """Seeded weights and compressed indexer keys for `n_layers` Memory-Indexer layers on top of an
    LsaWorkload (which supplies h_t, Dh, n_csa, C).  Shapes the paper leaves open (R28) are parameters:
    d_c (paper: r = 2048), c_I = 128, n_h = 64.  All arrays are stored bf16 bit patterns, transposed
    [out][in] (oracle/l1_oracle.py reading L1).

    Structure (the generator never evaluates Eq.(1)-(4): every quantity below is placed, not computed from the tower):
    W_w is built so that w = W_w h is about +1 on `n_pos` heads and -0.5 on the others, so random keys score clearly
    below the threshold.  The W_iuq block of a positive head p is rank one, sqrt(c_I) * r_p (x) v_p with a seeded unit
    direction r_p (c_I) and v_p ~ N(0, 1/d_c): whatever the low-rank code c of Eq.(1) turns out to be, that head's query
    is (sqrt(c_I) v_p.c) r_p - along +-r_p, with a magnitude ~|N(0,1)| sqrt(c_I) like the other heads'.  In about
    `hot_frac` of the chunks one entry is hot_gain / sqrt(c_I) * r_p for a positive head p: it matches that head with
    hot_gain * (v_p.c), i.e. clearly above the threshold for the heads whose v_p.c comes out near +1, clearly below for
    the others, and near it in between - which is where the tolerance band of the parity tests is exercised."""

    def __init__(self, wl: "LsaWorkload", n_layers: int = 3, d_c: int = 256, c_I: int = 128, n_h: int = 64, n_pos: int = 8,
                 hot_frac: float = 0.06, hot_gain: float = 14.0, tag: int = 900):
        c = wl.cfg
        assert c.dtype == "bf16"
        self.n_layers, self.d_c, self.c_I, self.n_h = n_layers, d_c, c_I, n_h
        self.layers: List[dict] = []
        self.index_k: List[List[np.ndarray]] = [[] for _ in range(c.B)]
        self.hot_chunks: List[List[np.ndarray]] = [[] for _ in range(c.B)]
        s = c.seed
        for l in range(n_layers):
            W_dq = _randn_stored(_rng(s, tag, l, 1), (d_c, c.Dh), 1.0 / math.sqrt(c.Dh), "bf16")
            g = _rng(s, tag, l, 3)
            a = np.full(n_h, -0.5)
            pos_heads = np.sort(g.choice(n_h, size=n_pos, replace=False))
            a[pos_heads] = 1.0
            W_iuq = _rng(s, tag, l, 2).standard_normal((n_h * c_I, d_c)) / math.sqrt(d_c)
            r_dir = _unit_rows(g.standard_normal((n_pos, c_I)))                  # r_p
            v_dir = g.standard_normal((n_pos, d_c)) / math.sqrt(d_c)             # v_p
            for j, p_ in enumerate(pos_heads):
                W_iuq[p_ * c_I:(p_ + 1) * c_I] = math.sqrt(c_I) * np.outer(r_dir[j], v_dir[j])
            W_iuq = store(W_iuq.astype(np.float32), "bf16")
            # one W_w for all sequences: built from the mean direction of the sequences' h0
            hbar = np.mean([as_f64(wl.h0[b], "bf16") for b in range(c.B)], axis=0)
            W_w = np.outer(a, hbar) / float(hbar @ hbar) + 0.02 * g.standard_normal((n_h, c.Dh)) / math.sqrt(c.Dh)
            W_w = store(W_w.astype(np.float32), "bf16")
            self.layers.append(dict(W_dq=W_dq, W_iuq=W_iuq, W_w=W_w))
            for b in range(c.B):
                n, nch = c.n_csa(b), c.n_chunks(b)
                gk = _rng(s, tag, l, 10 + b + c.seq_offset)
                K = gk.standard_normal((n, c_I)) / math.sqrt(c_I)
                hot = np.nonzero(gk.random(nch) < hot_frac)[0]
                for ch in hot:
                    lo, hi = ch * c.C, min(n, (ch + 1) * c.C)
                    e = int(gk.integers(lo, hi))
                    j = int(gk.integers(n_pos))
                    K[e] = hot_gain / math.sqrt(c_I) * r_dir[j]
                self.index_k[b].append(store(K.astype(np.float32), "bf16"))
                self.hot_chunks[b].append(hot)


class L2Inputs:
    """Seeded inputs of Level 2 (the native Lightning Indexer inside the resident set, Eq.(6)) on top of
    an LsaWorkload: one layer's compressed indexer keys per sequence, and per decode step the indexer queries
    q_idx [B][n_h][c_I] (bf16) and head weights w_idx [B][n_h] (fp32) of the token being decoded - inputs of the
    path like q (oracle/l2_oracle.py reading M3).  Keys and queries are N(0,1)/sqrt(sqrt(c_I)) each, so a
    per-head match is ~N(0,1); weights are N(0.5, 1)/n_h (mostly positive, some negative heads)."""

    def __init__(self, wl: "LsaWorkload", c_I: int = 128, n_h: int = 64, tag: int = 1200):
        c = wl.cfg
        assert c.dtype == "bf16"
        self.cfg, self.c_I, self.n_h, self.tag = c, c_I, n_h, tag
        s = c_I ** -0.25
        self.index_k: List[np.ndarray] = [_randn_stored(_rng(c.seed, tag, 1, b), (c.n_csa(b), c_I), s, "bf16") for b in range(c.B)]

    def q_idx(self, step: int) -> np.ndarray:
        c = self.cfg
        return _randn_stored(_rng(c.seed, self.tag, 2, step), (c.B, self.n_h, self.c_I), self.c_I ** -0.25, "bf16")

    def w_idx(self, step: int) -> np.ndarray:
        c = self.cfg
        g = _rng(c.seed, self.tag, 3, step)
        return ((0.5 + g.standard_normal((c.B, self.n_h))) / self.n_h).astype(np.float32)


# --------------------------------------------------------------------------------------
# NEXT-4 second half: the compressed history grows during decode ("all actively
# decoded tokens' CSA chunks" are an always-resident tier).  Inputs only: the entries a model's
# CSA / HCA compressors would hand over, and the embedding row of every chunk they complete.
# --------------------------------------------------------------------------------------
class GrowthInputs:
    """Seeded stand-ins for what DeepSeek-V4's compressors emit while decoding (they need the model):

    * before decode step t (t > 0, t % csa_every == 0) one CSA entry (K row, V row) per sequence - csa_every = 4 is the
      paper's "4:1" reading (R4); * before step t (t > 0, t % hca_every == 0) one HCA entry - 128:1;
    * when an entry completes a chunk, that chunk's embedding row: a random unit row, or (with probability `hot_frac`) a
      row planted at cosine `needle_cos` with the sequence's query direction, so that some completed chunks are recalled
      again later and their exported cold copy is really read.
    Capacities are what the caller must allocate: `cap_csa(b)` entries, `cap_hca(b)` rows."""

    def __init__(self, wl: "LsaWorkload", steps: int, csa_every: int = 4, hca_every: int = 128, hot_frac: float = 0.5,
                 tag: int = 1300):
        self.wl, self.steps, self.csa_every, self.hca_every, self.hot_frac, self.tag = wl, steps, csa_every, hca_every, hot_frac, tag

    def cap_csa(self, b: int) -> int:
        c = self.wl.cfg
        n = c.n_csa(b) + self.steps // self.csa_every + 1
        return -(-n // c.C) * c.C                      # whole chunks: the cold pool is allocated in pages

    def cap_hca(self, b: int) -> int:
        return self.wl.cfg.n_hca(b) + self.steps // self.hca_every + 1

    def csa_due(self, step: int) -> bool:
        return step > 0 and step % self.csa_every == 0

    def hca_due(self, step: int) -> bool:
        return step > 0 and step % self.hca_every == 0

    def csa_entry(self, step: int) -> Tuple[np.ndarray, np.ndarray]:
        """(K [B, D], V [B, D]) stored dtype: the entry handed over before decode step `step`."""
        c = self.wl.cfg
        g = _rng(c.seed, self.tag, 1, step)
        s = 1.0 / math.sqrt(c.D)
        return _randn_stored(g, (c.B, c.D), s, c.dtype), _randn_stored(g, (c.B, c.D), s, c.dtype)

    def hca_entry(self, step: int) -> Tuple[np.ndarray, np.ndarray]:
        c = self.wl.cfg
        g = _rng(c.seed, self.tag, 2, step)
        s = 1.0 / math.sqrt(c.D)
        return _randn_stored(g, (c.B, c.D), s, c.dtype), _randn_stored(g, (c.B, c.D), s, c.dtype)

    def emb_row(self, b: int, chunk: int) -> np.ndarray:
        """Embedding row [E] (stored dtype) of the chunk with id `chunk` of sequence b, handed over when it completes."""
        c = self.wl.cfg
        g = _rng(c.seed, self.tag, 3, b + c.seq_offset, chunk)
        r = g.standard_normal((1, c.E))
        if g.uniform() < self.hot_frac:
            row = LsaWorkload._plant(self.wl.u[b], r, np.full(1, c.needle_cos))
        else:
            row = _unit_rows(r)
        return store(row[0].astype(np.float32), c.dtype)


# --------------------------------------------------------------------------------------
# FP8 cold pool (NEXT-4 "FP8 KV pages", the host-link half): seeded e4m3 CODES and block scales.  Inputs only - the
# generator draws bytes, it never encodes or decodes a value (that arithmetic is the kernels' and the oracle's).
# --------------------------------------------------------------------------------------
class Fp8ColdInputs:
    """Per sequence: codes uint8 [n_chunks][2][C][D] and scales float32 [n_chunks][2] (K block, V block).

    A code byte is sign(1) | exponent(4) | mantissa(3).  Bytes are drawn so that the decoded magnitudes look like what a
    quantiser leaves of Gaussian rows: exponent fields concentrated in the top binades (field 15 - g, g geometric with
    p = 1/2, clipped at 0 = subnormals), uniform mantissa and sign; the NaN pattern (field 15, mantissa 7) is redrawn as
    mantissa 6.  Scales are powers of two 2^(-12 - (c mod 3)) (magnitudes around 1/sqrt(D) for D = 512), different per
    chunk and block so that a wrong scale index shows.  cfg 4/5-sized pools tile a base block like LsaWorkload does."""

    def __init__(self, wl: "LsaWorkload", tag: int = 1400):
        c = wl.cfg
        self.codes: List[np.ndarray] = []
        self.scales: List[np.ndarray] = []
        base = None
        if c.kv_base_chunks > 0:
            base = self._draw(_rng(c.seed, tag, 0), (c.kv_base_chunks, 2, c.C, c.D))
        for b in range(c.B):
            nch, gb = c.n_chunks(b), b + c.seq_offset
            if base is None:
                codes = self._draw(_rng(c.seed, tag, 1, gb), (nch, 2, c.C, c.D))
            else:
                idx = (np.arange(nch, dtype=np.int64) * 7 + 13 * gb) % c.kv_base_chunks
                codes = base[idx].copy()
                codes[:, 0, 0, 0] = (np.arange(nch) % 120 + 1).astype(np.uint8)      # a unique tag per chunk (a wrong copy shows)
            tail = nch * c.C - c.n_csa(b)
            if tail:
                codes[nch - 1, :, c.C - tail:, :] = 0                               # rows past n_csa: zero
            sc = np.empty((nch, 2), dtype=np.float32)
            sc[:, 0] = 2.0 ** (-12.0 - (np.arange(nch) % 3))
            sc[:, 1] = 2.0 ** (-12.0 - ((np.arange(nch) + 1) % 3))
            self.codes.append(codes)
            self.scales.append(sc)

    @staticmethod
    def _draw(g: np.random.Generator, shape) -> np.ndarray:
        n = int(np.prod(shape))
        expo = 15 - np.minimum(g.geometric(0.5, size=n) - 1, 15)
        mant = g.integers(0, 8, size=n)
        mant = np.where((expo == 15) & (mant == 7), 6, mant)
        sign = g.integers(0, 2, size=n)
        return ((sign << 7) | (expo << 3) | mant).astype(np.uint8).reshape(shape)
