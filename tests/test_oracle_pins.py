"""Pins for the CPU oracle: each function of oracle/lsa_oracle.py is checked against
something other than itself - hand-derived closed forms (tests/golden/hand_cases.json),
brute force on tiny inputs, invariants, special cases that reduce to a textbook / library
routine (torch float64 SDPA, cosine_similarity), and an independently structured LRU model.
PAPER.md prints no worked numeric example for this path, so no paper-printed values exist.
"""
import itertools
import json
import math
import os

import numpy as np
import pytest
import torch

from oracle import (LsaOracle, PoolExhausted, ResidencyOracle, attention, chunk_scores,
                    merge_partials, partial_attention, query_tower, topk_select, trigger_fires,
                    validate_selection, widen)
from paper_2606_09079_b200.workloads import (LsaWorkload, as_f64, make_config, make_small_config,
                                             plant_boundary_ties, store)
from lsa_harness import apply_emb_updates, make_oracle

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "hand_cases.json")))


# ---------------------------------------------------------------- O1 trigger
@pytest.mark.parametrize("tau,n,expect", [(64, 128, 2), (64, 2048, 32), (16, 1024, 64), (64, 1024, 16), (7, 50, 8)])
def test_trigger_closed_form(tau, n, expect):
    fired = [t for t in range(n) if trigger_fires(t, tau)]
    assert fired == list(range(0, n, tau))          # exactly {0, tau, 2tau, ...}
    assert len(fired) == expect == math.ceil(n / tau)


def test_trigger_stagger_cfg4():
    c = make_config(4)
    firsts = []
    for b in range(c.B):
        first = next(g for g in range(c.tau) if trigger_fires(c.step0(b) + g, c.tau))
        firsts.append(first)
        assert first == (b * c.tau // c.B) % c.tau    # R26: seq b first fires at global step 2b
    assert firsts == [2 * b for b in range(32)]


# ---------------------------------------------------------------- O2/O3 indexer
def test_indexer_hand_case():
    g = GOLD["indexer_3_4_5"]
    W, h, emb = (np.array(g[k], dtype=np.float32) for k in ("W_q", "h", "chunk_emb"))
    qh = query_tower(W, h)
    np.testing.assert_allclose(qh, g["q_hat"], rtol=0, atol=1e-15)
    # fp32 storage of 0.6/0.8 is inexact: compare at fp32 input-rounding level
    np.testing.assert_allclose(chunk_scores(qh, emb), g["scores"], rtol=0, atol=1e-7)
    assert topk_select(chunk_scores(qh, emb), 3)[0].tolist() == g["top3"]
    assert topk_select(chunk_scores(qh, emb), 2)[0].tolist() == g["top2"]


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_scores_match_planted_cosines(dtype):
    """Closed form: h0 is built (by least squares) so that W h0 is parallel to u, and
    Emb[c] = cos_c u + sqrt(1-cos_c^2) r_perp, hence score_c = cos_c up to input rounding."""
    wl = LsaWorkload(make_small_config(dtype, E=64, Dh=256, L=[65536, 65536], C=16), build_kv=False)
    tol = 2e-6 if dtype == "f32" else 1.5e-2
    for b in range(wl.cfg.B):
        qh = query_tower(wl.W_q, wl.h0[b])
        assert abs(np.linalg.norm(qh) - 1.0) < 1e-12
        assert float(qh @ wl.u[b]) > 1 - tol           # query tower lands on the planted direction
        sc = chunk_scores(qh, wl.base_emb[b])
        np.testing.assert_allclose(sc, wl.base_cos[b], atol=tol)
        ids = wl.needle_ids(b, 0)
        scn = chunk_scores(qh, wl.chunk_emb(b, 0))
        np.testing.assert_allclose(scn[ids], wl.cfg.needle_cos, atol=tol)


def test_scores_reduce_to_library_cosine():
    """score_c = cos(W h, Emb_c) * ||Emb_c||  via torch's cosine_similarity (library routine)."""
    g = np.random.default_rng(0)
    W = g.standard_normal((24, 40)).astype(np.float32)
    h = g.standard_normal(40).astype(np.float32)
    emb = g.standard_normal((50, 24)).astype(np.float32)
    z = torch.from_numpy(W).double() @ torch.from_numpy(h).double()
    e = torch.from_numpy(emb).double()
    ref = torch.nn.functional.cosine_similarity(z[None, :], e, dim=1) * e.norm(dim=1)
    np.testing.assert_allclose(chunk_scores(query_tower(W, h), emb), ref.numpy(), rtol=1e-12, atol=1e-13)


def test_indexer_invariants():
    g = np.random.default_rng(1)
    W = g.standard_normal((16, 32)).astype(np.float32)
    h = g.standard_normal(32).astype(np.float32)
    qh = query_tower(W, h)
    np.testing.assert_allclose(query_tower(W, 4 * h), qh, atol=1e-15)      # scale invariance in h
    np.testing.assert_allclose(query_tower(W, -h), -qh, atol=1e-15)        # odd in h (sign kept)
    assert abs(chunk_scores(qh, qh[None, :].astype(np.float64))[0] - 1.0) < 1e-12   # Emb = q_hat -> 1
    perp = g.standard_normal(16); perp -= (perp @ qh) * qh
    assert abs(chunk_scores(qh, perp[None, :])[0]) < 1e-12                 # orthogonal -> 0
    z0 = query_tower(W, np.zeros(32, dtype=np.float32))                    # R16: zero-norm clamp
    assert np.all(z0 == 0) and np.all(np.isfinite(z0))
    assert topk_select(chunk_scores(z0, g.standard_normal((9, 16))), 4)[0].tolist() == [0, 1, 2, 3]
    # transposed-operand mistake would fail here: non-square W with distinct row/col structure
    W2 = np.zeros((2, 3), dtype=np.float32); W2[0, 2] = 1; W2[1, 0] = 1
    np.testing.assert_allclose(query_tower(W2, np.array([3, 9, 4], dtype=np.float32)), [0.8, 0.6], atol=1e-15)


# ---------------------------------------------------------------- O4 top-k
def _brute_topk(scores, k):
    order = sorted(range(len(scores)), key=lambda c: (-float(scores[c]), c))
    return order[: min(k, len(scores))]


def test_topk_brute_force_all_k():
    g = np.random.default_rng(2)
    for n in (1, 2, 5, 17, 64):
        for trial in range(6):
            sc = g.standard_normal(n)
            if trial % 2:                                    # force duplicates
                sc = np.round(sc * 2) / 2
            for k in range(1, n + 3):
                sel, val = topk_select(sc, k)
                bf = _brute_topk(sc, k)
                assert sel[: len(bf)].tolist() == bf
                assert np.all(sel[len(bf):] == -1) and np.all(val[len(bf):] == -np.inf)
                np.testing.assert_array_equal(val[: len(bf)], sc[bf])


def test_topk_all_equal_and_permutations():
    assert topk_select(np.full(10, 0.25), 4)[0].tolist() == [0, 1, 2, 3]
    for perm in itertools.permutations([0.1, 0.5, 0.5, -2.0]):
        sc = np.array(perm)
        assert topk_select(sc, 3)[0].tolist() == _brute_topk(sc, 3)


def test_validate_selection_rules():
    sc = np.array([0.9, 0.5, 0.5, 0.5 * (1 + 5e-6), 0.1, 0.5])
    assert validate_selection(np.array([0, 3, 1]), sc, 3) is None
    assert validate_selection(np.array([0, 1, 3]), sc, 3) is None          # in-band order swap allowed
    assert validate_selection(np.array([0, 1, 2]), sc, 3) is None          # in-band substitution allowed
    assert "tie-break" in validate_selection(np.array([0, 3, 2]), sc, 3)   # exact tie: lower id must win
    assert "missing" in validate_selection(np.array([1, 2, 3]), sc, 3)
    assert "below" in validate_selection(np.array([0, 3, 4]), sc, 3)
    assert "duplicate" in validate_selection(np.array([0, 3, 3]), sc, 3)
    assert validate_selection(np.array([0, 3, 1, 2, 5, 4, -1, -1]), sc, 8) is None
    assert "padding" in validate_selection(np.array([0, 3, 1, 2, 5, 4, 0, -1]), sc, 8)


# ---------------------------------------------------------------- O6 attention
def test_attention_hand_case():
    g = GOLD["attention_two_keys"]
    out, lse, p = attention(np.array(g["q"]), np.array(g["K"]), np.array(g["V"]), g["sm_scale"])
    np.testing.assert_allclose(p, g["p"], atol=1e-15)
    np.testing.assert_allclose(out, g["out"], atol=1e-14)
    np.testing.assert_allclose(lse, g["lse"], atol=1e-15)


def test_attention_special_cases():
    g = np.random.default_rng(3)
    H, D, N = 5, 16, 37
    q, K, V = g.standard_normal((H, D)), g.standard_normal((N, D)), g.standard_normal((N, D))
    out1, lse1, p1 = attention(q, K[:1], V[:1], 0.3)
    np.testing.assert_array_equal(out1, np.broadcast_to(V[0], (H, D)))      # single key -> its value
    np.testing.assert_allclose(lse1, 0.3 * (q @ K[0]), atol=1e-14)
    outm, _, pm = attention(q, np.broadcast_to(K[3], (N, D)), V, 0.3)        # equal keys -> mean(V)
    np.testing.assert_allclose(outm, np.broadcast_to(V.mean(0), (H, D)), atol=1e-13)
    out, lse, p = attention(q, K, V, 0.3)
    assert np.all(np.abs(p.sum(1) - 1.0) < 1e-12) and np.all(p >= 0)        # weights sum to 1
    assert np.all(out <= V.max(0) + 1e-12) and np.all(out >= V.min(0) - 1e-12)   # convex combination
    perm = g.permutation(N)                                                  # key-order invariance
    outp, lsep, _ = attention(q, K[perm], V[perm], 0.3)
    np.testing.assert_allclose(outp, out, atol=1e-13); np.testing.assert_allclose(lsep, lse, atol=1e-13)
    oute, lsee, _ = attention(q, K[:0], V[:0], 0.3)                          # empty key set
    assert np.all(oute == 0) and np.all(lsee == -np.inf)
    # shifting all logits by a constant leaves out unchanged and shifts lse (stability of max-subtraction)
    big = attention(q * 200, K, V, 1.0)[0]
    assert np.all(np.isfinite(big))


def test_attention_matches_torch_sdpa_fp64():
    g = np.random.default_rng(4)
    H, D, N = 8, 32, 300
    q, K, V = g.standard_normal((H, D)), g.standard_normal((N, D)), g.standard_normal((N, D))
    scale = 1 / math.sqrt(D)
    ref = torch.nn.functional.scaled_dot_product_attention(
        torch.from_numpy(q)[None], torch.from_numpy(K)[None].expand(1, N, D), torch.from_numpy(V)[None],
        scale=scale)[0].numpy()
    np.testing.assert_allclose(attention(q, K, V, scale)[0], ref, rtol=1e-12, atol=1e-13)


def test_merge_partials_any_partition():
    g = np.random.default_rng(5)
    H, D, N = 4, 8, 101
    q, K, V = g.standard_normal((H, D)) * 3, g.standard_normal((N, D)), g.standard_normal((N, D))
    out, lse, _ = attention(q, K, V, 0.7)
    for cuts in ([50], [1, 2, 3], [10, 40, 41, 100], list(range(1, N))):
        edges = [0] + cuts + [N]
        parts = [partial_attention(q, K[a:b], V[a:b], 0.7) for a, b in zip(edges[:-1], edges[1:])]
        o2, l2 = merge_partials(parts)
        np.testing.assert_allclose(o2, out, rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(l2, lse, rtol=1e-12, atol=1e-13)


# ---------------------------------------------------------------- O5 residency
def test_lru_hand_trace():
    g = GOLD["lru_trace"]
    r = ResidencyOracle(1, [g["n_chunks"]], g["hot_pages"])
    for step, call in enumerate(g["calls"]):
        fl = r.fetch(0, call["selection"], step, 0)
        assert [list(x) for x in fl] == call["fetch_list"]
        assert r.maybe_swap(0, step)
        assert [list(x) for x in r.cur[0]] == call["table"]
    fc = g["final_counters"]
    assert (r.hits, r.misses, r.evictions) == (fc["hits"], fc["misses"], fc["evictions"])


class _NaiveLru:
    """Independently structured model: one recency list (least -> most recent); never-used pages
    start in index order; pages touched in one call move to the back in page order."""

    def __init__(self, P):
        self.order = list(range(P))
        self.owner = {}

    def fetch(self, key_of, sel_up, pinned):
        touched, out = [], []
        for c in sel_up:
            if key_of(c) in self.owner.values():
                p = next(p for p, o in self.owner.items() if o == key_of(c))
                touched.append(p)
        pinned = set(pinned) | set(touched)
        for c in sel_up:
            if key_of(c) in self.owner.values():
                continue
            p = next(p for p in self.order if p not in pinned)
            self.owner[p] = key_of(c)
            pinned.add(p); touched.append(p); out.append((c, p))
        for p in sorted(touched):
            self.order.remove(p); self.order.append(p)
        return out


@pytest.mark.parametrize("seed", range(6))
def test_residency_vs_naive_lru_and_invariants(seed):
    g = np.random.default_rng(100 + seed)
    B, k, lag = 3, 3, seed % 2
    n_chunks = [7, 12, 5]
    P = 2 * B * k + (seed % 3)
    cold = [g.integers(0, 2**16, size=(n, 2, 4, 8), dtype=np.uint16) for n in n_chunks]
    r = ResidencyOracle(B, n_chunks, P, cold)
    naive = _NaiveLru(P)
    step = 0
    for it in range(40):
        for b in range(B):
            r.maybe_swap(b, step)
        fire = [b for b in range(B) if g.random() < 0.5]
        for b in fire:
            sel = g.choice(n_chunks[b], size=min(k, n_chunks[b]), replace=False)
            resident_before = {c for c in sel if r.page_of[b][c] >= 0}
            bytes_before, miss_before = r.bytes_fetched, r.misses
            pins = {p for bb in range(B) for _, p in r.cur[bb]} | \
                   {p for bb in range(B) if bb != b and r.nxt[bb] is not None for _, p in r.nxt[bb]}
            fl = r.fetch(b, sel, step, lag)
            assert fl == naive.fetch(lambda c: (b, c), sorted(int(c) for c in sel), pins)
            assert r.misses - miss_before == len(sel) - len(resident_before) == len(fl)
            assert r.bytes_fetched - bytes_before == len(fl) * cold[b][0].nbytes
            assert [c for c, _ in r.nxt[b]] == sorted(int(c) for c in sel)
            if lag == 0:
                r.maybe_swap(b, step)
        # invariants: owner / page_of mutually inverse, no page owned twice, bytes match cold pool
        seen = {}
        for p, o in enumerate(r.owner):
            if o is not None:
                assert o not in seen; seen[o] = p
                assert r.page_of[o[0]][o[1]] == p
                assert np.array_equal(r.hot[p], cold[o[0]][o[1]])
        for b in range(B):
            for c, p in enumerate(r.page_of[b]):
                assert p == -1 or r.owner[p] == (b, c)
            for c, p in r.cur[b] + (r.nxt[b] or []):
                assert r.owner[p] == (b, c)             # attended pages are always resident
        step += 1


def test_residency_big_pool_fetches_once_and_exhaustion():
    r = ResidencyOracle(1, [10], 10)
    g = np.random.default_rng(7)
    for step in range(30):
        r.maybe_swap(0, step)
        r.fetch(0, g.choice(10, size=3, replace=False), step, 1)
    assert r.misses <= 10 and r.evictions == 0           # P >= n_chunks: each chunk fetched at most once
    r2 = ResidencyOracle(1, [10], 3)
    r2.fetch(0, [0, 1], 0, 0); r2.maybe_swap(0, 0)
    with pytest.raises(PoolExhausted):
        r2.fetch(0, [2, 3], 1, 0)                        # cur pins 2 pages, only 1 left for 2 misses


# ---------------------------------------------------------------- the whole path
def test_full_path_cfg1_selects_needles_and_window_rule():
    wl = LsaWorkload(make_config(1))
    c = wl.cfg
    orc = make_oracle(wl)
    fetch_steps, outs = [], {}
    for t in range(c.steps):
        q = wl.q(t); kn, vn = wl.kv_new(t)
        before = orc.pool.bytes_fetched
        fired, (out, lse) = orc.run_step(q, wl.h(t), kn, vn)
        if orc.pool.bytes_fetched != before:
            fetch_steps.append(t)
        if fired:
            assert sorted(fired[0][0].tolist()) == wl.needle_ids(0, 0).tolist()   # the 4 planted needles
            np.testing.assert_allclose(fired[0][1], c.needle_cos, atol=1e-2)    # h_t = h0 + 0.05*eps drifts off u a little
        outs[t] = out
        assert np.all(np.isfinite(out))
    assert fetch_steps == [0]            # P:185 zero transfers inside a window; static scores -> no refetch
    assert orc.pool.triggers == 2 and orc.pool.misses == 4 and orc.pool.hits == 4


def test_recall_lag_visibility():
    """attention at the trigger step uses the old table, step t+1 the new one."""
    wl = LsaWorkload(make_small_config("f32", B=1, L=[4096], tau=4, k=3, hot_pages=8))
    for lag in (0, 1, 3):
        orc = make_oracle(wl, recall_lag=lag)
        sizes = []
        for t in range(6):
            orc.run_step(wl.q(t), wl.h(t))
            sizes.append(len(orc.pool.cur[0]))
        assert sizes == [0] * lag + [3] * (6 - lag)          # visible from step t + lag on
    # direct check that the table used at the trigger step is the OLD one
    orc = make_oracle(wl, recall_lag=1)
    orc.step_begin(wl.h(0))
    K, _ = orc.gather_kv(0)
    assert K.shape[0] == wl.cfg.n_hca(0) + wl.cfg.W          # HCA + window only at step 0


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_k_equals_all_chunks_is_dense_attention(dtype):
    """BJ north_star self-check / P:185 'byte-identical to baseline': with k = n_chunks and
    P >= n_chunks the path equals textbook dense attention over HCA + all CSA + window."""
    cfg = make_small_config(dtype, B=2, L=[2048, 1216], k=32, hot_pages=64, recall_lag=0, tau=4, q_gain=8.0)
    wl = LsaWorkload(cfg)
    orc = make_oracle(wl)
    q = wl.q(0)
    _, (out, lse) = orc.run_step(q, wl.h(0))
    for b in range(cfg.B):
        assert len(orc.pool.cur[b]) == cfg.n_chunks(b) < 32 or cfg.n_chunks(b) == 32
        ncsa = cfg.n_csa(b)
        cold = as_f64(wl.cold_csa[b], dtype)
        Kd = np.concatenate([as_f64(wl.hca_k[b], dtype), cold[:, 0].reshape(-1, cfg.D)[:ncsa], as_f64(wl.win_k[b], dtype)])
        Vd = np.concatenate([as_f64(wl.hca_v[b], dtype), cold[:, 1].reshape(-1, cfg.D)[:ncsa], as_f64(wl.win_v[b], dtype)])
        ref = torch.nn.functional.scaled_dot_product_attention(
            torch.from_numpy(as_f64(q[b], dtype))[None], torch.from_numpy(Kd)[None], torch.from_numpy(Vd)[None],
            scale=1 / math.sqrt(cfg.D))[0].numpy()
        np.testing.assert_allclose(out[b], ref, rtol=1e-11, atol=1e-13)


def test_needle_drift_and_selection_contains_needles_cfg3_indexer_only():
    """cfg 3 indexer at full size (no K/V built): every trigger's top-64 contains the 16 needles."""
    wl = LsaWorkload(make_config(3), build_kv=False)
    c = wl.cfg
    emb = wl.chunk_emb(0, 0)
    for trig in range(0, 9):
        g = trig * c.tau
        upd = wl.emb_row_updates(0, trig)
        if upd is not None:
            emb = emb.copy(); emb[upd[0]] = upd[1]
            assert not np.array_equal(wl.needle_ids(0, trig), wl.needle_ids(0, trig - 1))
        np.testing.assert_array_equal(emb, wl.chunk_emb(0, trig))
        sc = chunk_scores(query_tower(wl.W_q, wl.h(g)[0]), emb)
        sel, val = topk_select(sc, c.k)
        assert set(wl.needle_ids(0, trig).tolist()) <= set(sel.tolist())
        assert len(set(sel.tolist())) == c.k


def test_planted_boundary_ties():
    wl = LsaWorkload(make_config(5, B=1, L=[524288]), build_kv=False)
    c = wl.cfg
    emb = wl.chunk_emb(0, 0)
    qh = query_tower(wl.W_q, wl.h(0)[0])
    order = topk_select(chunk_scores(qh, emb), c.n_chunks(0))[0]
    emb2 = plant_boundary_ties(emb, order, c.k, c.dtype)
    sc2 = chunk_scores(qh, emb2)
    a, b_, c_ = order[c.k - 1], order[c.k], order[c.k + 1]
    assert sc2[a] == sc2[b_]                                    # exact tie across the boundary
    assert 0 < abs(sc2[c_] - sc2[a]) < 1e-4                     # near tie
    sel = topk_select(sc2, c.k)[0]
    assert (min(a, b_) in sel) and (max(a, b_) not in sel)      # lower chunk id wins
