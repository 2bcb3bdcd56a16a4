"""Pins for oracle/l2_oracle.py (Level 2: native Lightning-Indexer Top-k inside the resident set, Eq.(6)).
Each function is checked against something other than itself: a hand-computed case (tests/golden/l2_hand_case.json),
brute force, invariants, the relation to the independently pinned Level-1 oracle (Eq.(4) = sigmoid of the native
score), and special cases that reduce to the already pinned Level-1-only path (k2 >= all resident entries ->
LsaOracle.decode_attention; k2 = 0 -> attention over HCA (+) window only)."""
import itertools
import json
import os

import numpy as np
import pytest

from oracle import attention, widen
from oracle.l1_oracle import l1_entry_scores
from oracle.l2_oracle import (l2_decode_attention, l2_gather_kv, l2_native_scores, l2_resident_entries, l2_select,
                              l2_topk_entries, validate_l2_selection)
from paper_2606_09079_b200.workloads import L2Inputs, LsaWorkload, make_small_config
from lsa_harness import make_oracle

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "l2_hand_case.json")))


def test_hand_case():
    g = GOLD
    q, w, K = (np.array(g[k], dtype=np.float32) for k in ("q_idx", "w_idx", "index_k"))
    np.testing.assert_array_equal(l2_native_scores(q, w, K), g["scores_all"])
    ids = l2_resident_entries(g["table_chunks"], g["n_csa"], g["C"])
    assert ids.tolist() == g["resident_entries"]                       # partial chunk 3 contributes one row (M1)
    for k2, key in ((3, "top3"), (1, "top1"), (9, "top9")):
        sel, ids2, sc = l2_select(q, w, K, g["table_chunks"], g["n_csa"], g["C"], k2)
        assert sel.tolist() == g[key]
        assert ids2.tolist() == g["resident_entries"]
        np.testing.assert_array_equal(sc, [g["scores_all"][i] for i in g["resident_entries"]])
    assert l2_select(q, w, K, g["table_chunks"], g["n_csa"], g["C"], 0)[0].tolist() == []
    assert l2_select(q, w, K, [], g["n_csa"], g["C"], 4)[0].tolist() == []


def test_native_score_is_eq4_without_sigmoid_and_invariants():
    g = np.random.default_rng(5)
    q = g.standard_normal((6, 8)).astype(np.float32)
    w = g.standard_normal(6)
    K = g.standard_normal((40, 8)).astype(np.float32)
    s = l2_native_scores(q, w, K)
    I, pre = l1_entry_scores(widen(q), w, K)                           # Level-1 oracle, pinned on its own
    np.testing.assert_allclose(s, pre, rtol=0, atol=1e-13)
    np.testing.assert_allclose(1.0 / (1.0 + np.exp(-s)), I, rtol=0, atol=1e-13)
    # per-entry brute force, written as loops
    for e in (0, 7, 39):
        acc = 0.0
        for h in range(6):
            d = sum(float(q[h, j]) * float(K[e, j]) for j in range(8))
            acc += w[h] * (d if d > 0 else 0.0)
        assert abs(acc - s[e]) < 1e-12
    np.testing.assert_allclose(l2_native_scores(q, 3.0 * w, K), 3.0 * s, atol=1e-12)       # linear in w
    perm = g.permutation(6)
    np.testing.assert_allclose(l2_native_scores(q[perm], w[perm], K), s, atol=1e-12)       # head order is irrelevant
    np.testing.assert_allclose(l2_native_scores(2.0 * q, w, K), 2.0 * s, atol=1e-12)       # ReLU is positively homogeneous
    # the gate matters: with one head, w = 1, the score is max(q.K, 0) - never negative, zero where q.K < 0
    s1 = l2_native_scores(q[:1], np.ones(1), K)
    d1 = widen(K) @ widen(q[0])
    assert (s1 >= 0).all() and np.array_equal(s1 == 0, d1 <= 0) and np.allclose(s1[d1 > 0], d1[d1 > 0])
    # a negative head weight subtracts
    assert np.allclose(l2_native_scores(q[:1], -np.ones(1), K), -s1)


def test_topk_brute_force_with_ties():
    g = np.random.default_rng(11)
    for n in (1, 2, 5, 9):
        for trial in range(20):
            sc = g.integers(0, 4, size=n).astype(np.float64)           # many exact ties
            ids = np.sort(g.choice(50, size=n, replace=False))
            for k2 in range(0, n + 2):
                got = l2_topk_entries(sc, ids, k2).tolist()
                m = min(k2, n)
                assert len(got) == m
                # brute force: the chosen SET is the one subset of size m no outsider beats (score desc, id asc)
                best = None
                for sub in itertools.combinations(range(n), m):
                    inside = set(sub)
                    ok = all((sc[i], -ids[i]) >= (sc[o], -ids[o]) for i in inside for o in range(n) if o not in inside)
                    if ok:
                        assert best is None                                # unique because ids are
                        best = sorted(sub, key=lambda j: (-sc[j], ids[j]))
                assert got == [int(ids[j]) for j in best]


def _small(k2_frac=None):
    cfg = make_small_config("bf16", steps=2, q_gain=8.0)
    wl = LsaWorkload(cfg)
    orc = make_oracle(wl)
    orc.run_step(wl.q(0), wl.h(0), *wl.kv_new(0))                       # trigger at step 0 (recall_lag decides visibility)
    orc.run_step(wl.q(1), wl.h(1), *wl.kv_new(1))
    return cfg, wl, orc


def test_k2_covering_everything_is_the_level1_only_path():
    cfg, wl, orc = _small()
    l2 = L2Inputs(wl, c_I=16, n_h=4)
    q = wl.q(2)
    ref_out, ref_lse = orc.decode_attention(q)                           # pinned in tests/test_oracle_pins.py
    sels = []
    for b in range(cfg.B):
        chunks = [c for c, _ in orc.pool.cur[b]]
        assert chunks, "the staged table must be current by now"
        sel, ids, sc = l2_select(l2.q_idx(2)[b], l2.w_idx(2)[b], l2.index_k[b], chunks, cfg.n_csa(b), cfg.C, 10 ** 9)
        assert sorted(sel.tolist()) == ids.tolist()
        sels.append(sel)
    out, lse = l2_decode_attention(orc, q, sels)
    np.testing.assert_allclose(out, ref_out, rtol=0, atol=1e-12)
    np.testing.assert_allclose(lse, ref_lse, rtol=0, atol=1e-12)


def test_k2_zero_is_hca_plus_window_and_single_entry_case():
    cfg, wl, orc = _small()
    q = wl.q(2)
    out, lse = l2_decode_attention(orc, q, [[] for _ in range(cfg.B)])
    for b in range(cfg.B):
        K = np.concatenate([widen(orc.hca_k[b]), widen(orc.win_k[b][: orc.w_len[b]])])
        V = np.concatenate([widen(orc.hca_v[b]), widen(orc.win_v[b][: orc.w_len[b]])])
        o, l, _ = attention(widen(q[b]), K, V, orc.sm_scale)
        np.testing.assert_allclose(out[b], o, atol=1e-13)
        # one selected entry: its K/V rows are exactly row r of the page its chunk occupies (M1), placed between HCA and window
        c, p = orc.pool.cur[b][0]
        s = c * cfg.C + 3
        Kg, Vg = l2_gather_kv(orc, b, [s])
        n_hca = len(orc.hca_k[b])
        assert Kg.shape[0] == n_hca + 1 + orc.w_len[b]
        np.testing.assert_array_equal(Kg[n_hca], widen(orc.pool.hot[p][0, 3]))
        np.testing.assert_array_equal(Vg[n_hca], widen(orc.pool.hot[p][1, 3]))
        np.testing.assert_array_equal(Kg[n_hca], widen(wl.cold_csa[b][c][0, 3]))      # and of the cold mirror (fetch is a copy)


def test_selection_only_from_resident_valid_rows_and_validator():
    cfg, wl, orc = _small()
    l2 = L2Inputs(wl, c_I=16, n_h=4)
    b = 0
    chunks = [c for c, _ in orc.pool.cur[b]]
    sel, ids, sc = l2_select(l2.q_idx(2)[b], l2.w_idx(2)[b], l2.index_k[b], chunks, cfg.n_csa(b), cfg.C, 7)
    assert len(sel) == 7 and set(sel.tolist()) <= set(ids.tolist())
    assert all((s // cfg.C) in chunks and s < cfg.n_csa(b) for s in sel.tolist())
    full = l2_native_scores(l2.q_idx(2)[b], l2.w_idx(2)[b], l2.index_k[b])
    np.testing.assert_allclose(sc, full[ids], atol=1e-12)                             # restriction of the full scan
    assert min(full[s] for s in sel.tolist()) >= max(full[i] for i in ids.tolist() if i not in set(sel.tolist()))
    padded = np.full(10, -1); padded[:7] = sel
    assert validate_l2_selection(padded, ids, sc, 7) is None
    bad = padded.copy(); bad[6] = [i for i in ids.tolist() if i not in set(sel.tolist())][-1]
    ranked = sorted(ids.tolist(), key=lambda e: (-full[e], e))
    bad[6] = ranked[-1]                                                                 # the worst entry instead of the 7th
    assert validate_l2_selection(bad, ids, sc, 7) is not None
    assert validate_l2_selection(padded[:6], ids, sc, 7) is not None                    # too few
    # a swap inside the tolerance band is accepted, outside it is not
    sc2 = np.array([5.0, 4.0, 3.0, 3.0 - 1e-7, 1.0]); ids2 = np.arange(5)
    assert validate_l2_selection([0, 1, 3], ids2, sc2, 3) is None
    assert validate_l2_selection([0, 1, 4], ids2, sc2, 3) is not None


def test_l2_inputs_are_seeded_and_shaped():
    """The Level-2 input generator holds none of the method's arithmetic: shapes, determinism and the stated distributions."""
    cfg = make_small_config("bf16", steps=2)
    wl = LsaWorkload(cfg, build_kv=False)
    a, b = L2Inputs(wl, c_I=16, n_h=4), L2Inputs(wl, c_I=16, n_h=4)
    for x, y in zip(a.index_k, b.index_k):
        assert x.dtype == np.uint16 and np.array_equal(x, y)
    assert [k.shape for k in a.index_k] == [(cfg.n_csa(i), 16) for i in range(cfg.B)]
    assert np.array_equal(a.q_idx(3), b.q_idx(3)) and not np.array_equal(a.q_idx(3), a.q_idx(4))
    assert a.q_idx(0).shape == (cfg.B, 4, 16) and a.w_idx(0).shape == (cfg.B, 4) and a.w_idx(0).dtype == np.float32
    big = L2Inputs(wl, c_I=128, n_h=64)
    w = np.concatenate([big.w_idx(t).ravel() for t in range(40)])
    assert abs(w.mean() * 64 - 0.5) < 0.1 and abs(w.std() * 64 - 1.0) < 0.1
    m = widen(big.index_k[0][:512]) @ widen(big.q_idx(0)[0]).T              # per-head matches ~ N(0, 1)
    assert abs(m.std() - 1.0) < 0.1 and abs(m.mean()) < 0.05
