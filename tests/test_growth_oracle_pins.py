"""Pins for oracle/growth_oracle.py (NEXT-4 second half, R29-R33).  CPU only.

Each pin ties the growth oracle to something other than itself: the plain dense definition of attention over
the grown history, the STATIC oracle initialised with the longer history, a schedule traced by hand
(tests/golden/growth_hand_case.json), and invariants of the rules the readings state."""
import json
import math
import os

import numpy as np
import pytest

from oracle import LsaOracle, attention, widen
from oracle.growth_oracle import TIER_SLOTS, GrowingLsaOracle, TierOverflow
from paper_2606_09079_b200.workloads import GrowthInputs, LsaWorkload, make_small_config

from lsa_harness import make_growing_oracle, oracle_appends

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def tiny_oracle(*, C, n_csa0, cap_chunks, k, tau, lag, hot_pages, D=4, H=2, W=3, E=4, Dh=6, n_hca0=1, cap_hca=4, seed=5):
    g = np.random.default_rng(seed)
    cold = np.zeros((cap_chunks, 2, C, D), dtype=np.float32)
    flat = g.standard_normal((n_csa0, 2, D)).astype(np.float32)          # entry s -> (K row, V row)
    for s in range(n_csa0):
        cold[s // C, 0, s % C], cold[s // C, 1, s % C] = flat[s, 0], flat[s, 1]
    emb = np.zeros((cap_chunks, E), dtype=np.float32)
    emb[: n_csa0 // C] = g.standard_normal((n_csa0 // C, E))
    hk, hv = np.zeros((cap_hca, D), np.float32), np.zeros((cap_hca, D), np.float32)
    hk[:n_hca0], hv[:n_hca0] = g.standard_normal((n_hca0, D)), g.standard_normal((n_hca0, D))
    orc = GrowingLsaOracle(dtype="f32", H=H, D=D, C=C, W=W, k=k, tau=tau, recall_lag=lag, hot_pages=hot_pages,
                           W_q=g.standard_normal((E, Dh)).astype(np.float32), cold_csa=[cold], n_csa=[n_csa0], n_hca=[n_hca0],
                           chunk_emb=[emb], hca_k=[hk], hca_v=[hv], win_k=[g.standard_normal((W, D)).astype(np.float32)],
                           win_v=[g.standard_normal((W, D)).astype(np.float32)], w_len=[W], w_head=[0], step0=[0])
    return orc, g, [tuple(x) for x in flat]


def test_hand_traced_tier_schedule():
    """Every quantity of the hand trace: candidates, tier membership, what each trigger sees, exports, tier pages."""
    hc = json.load(open(os.path.join(GOLDEN, "growth_hand_case.json")))
    C, k = hc["C"], 4
    orc, g, _ = tiny_oracle(C=C, n_csa0=hc["n_csa0"], cap_chunks=8, k=k, tau=hc["tau"], lag=hc["recall_lag"], hot_pages=8)
    assert orc.P_lru == 8 - TIER_SLOTS and orc.k_sel == k - TIER_SLOTS
    seen = []
    for t in range(hc["steps"]):
        if t > 0 and t % hc["csa_every"] == 0:
            before = orc.exported
            orc.append_compressed(0, g.standard_normal(4).astype(np.float32), g.standard_normal(4).astype(np.float32),
                                  emb_row=g.standard_normal(4).astype(np.float32))
            if str(t) in hc["exported_chunks_by_step"]:
                assert orc.exported == before + 1 and orc.n_chunks[0] - 1 == hc["exported_chunks_by_step"][str(t)]
            else:
                assert orc.exported == before
        fired = orc.step_begin(g.standard_normal((1, 6)).astype(np.float32))
        if fired:
            seen.append(orc.ncand_nxt[0])
            assert t in hc["trigger_steps"]
        assert orc.n_csa[0] == hc["n_csa"][t], t
        assert orc.n_chunks[0] == hc["candidates"][t], t
        assert orc.tier(0) == hc["tier"][t], (t, orc.tier(0))
        tbl = orc.table(0)
        n_sel = len(orc.pool.cur[0])
        assert [c for c, _ in tbl[n_sel:]] == hc["tier"][t]
        for c, p in tbl[n_sel:]:
            assert p == orc.P_lru + hc["tier_page_offset"][str(c)]
        assert [c for c, _ in tbl] == sorted(c for c, _ in tbl)                   # R13 still holds
        orc.step_end(g.standard_normal((1, 2, 4)).astype(np.float32), attend=False)
    assert seen == hc["candidates_seen_by_trigger"]


def test_third_tier_chunk_is_refused():
    """R31: the tier holds two chunks; a chunk every 2 steps against tau = 3 overflows it (hand trace in DESIGN R31)."""
    orc, g, _ = tiny_oracle(C=2, n_csa0=4, cap_chunks=16, k=4, tau=3, lag=1, hot_pages=8)
    with pytest.raises(TierOverflow):
        for t in range(12):
            if t > 0:
                orc.append_compressed(0, np.zeros(4, np.float32), np.zeros(4, np.float32), emb_row=np.zeros(4, np.float32))
            orc.step_begin(g.standard_normal((1, 6)).astype(np.float32))
            orc.step_end(None, attend=False)


@pytest.mark.parametrize("lag", [0, 1])
def test_everything_recalled_equals_dense_attention_over_the_grown_history(lag):
    """With k_sel >= every chunk and a trigger every step, the attended set must be exactly: all HCA rows so far, ALL CSA
    entries so far (recalled full chunks + tier), the window.  Compared with the plain definition over arrays the TEST keeps
    itself (flat lists, no tables), and with a static LsaOracle initialised with the longer history."""
    C, D, H, W = 3, 4, 2, 3
    orc, g, flat = tiny_oracle(C=C, n_csa0=7, cap_chunks=12, k=12 + TIER_SLOTS, tau=1, lag=lag, hot_pages=2 * 12 + TIER_SLOTS,
                               D=D, H=H, W=W)
    hca = [(orc.hca_k[0][0].copy(), orc.hca_v[0][0].copy())]
    for t in range(20):
        if t > 0 and t % 2 == 0:
            kr, vr = g.standard_normal(D).astype(np.float32), g.standard_normal(D).astype(np.float32)
            orc.append_compressed(0, kr, vr, emb_row=g.standard_normal(4).astype(np.float32))
            flat.append((kr, vr))
        if t > 0 and t % 7 == 0:
            kr, vr = g.standard_normal(D).astype(np.float32), g.standard_normal(D).astype(np.float32)
            orc.append_compressed(0, hca_k=kr, hca_v=vr)
            hca.append((kr, vr))
        h = g.standard_normal((1, 6)).astype(np.float32)
        q = g.standard_normal((1, H, D)).astype(np.float32)
        kn, vn = g.standard_normal((1, D)).astype(np.float32), g.standard_normal((1, D)).astype(np.float32)
        orc.step_begin(h)
        # what SHOULD be attended at this step
        if lag == 1 and t == 0:
            csa_idx = [6]                                   # before the first table is visible: only the tier (R10 + R30)
        elif lag == 1:
            # the current table comes from the trigger one step ago: it holds the chunks that were full then; everything
            # started since is tier
            csa_idx = list(range(len(flat)))
        else:
            csa_idx = list(range(len(flat)))
        res, _ = orc.step_end(q, kn, vn)
        win_k, win_v = orc.win_k[0][: orc.w_len[0]], orc.win_v[0][: orc.w_len[0]]
        K = np.concatenate([np.stack([a for a, _ in hca]), np.stack([flat[s][0] for s in csa_idx]), win_k]).astype(np.float64)
        V = np.concatenate([np.stack([b for _, b in hca]), np.stack([flat[s][1] for s in csa_idx]), win_v]).astype(np.float64)
        want, _, _ = attention(q[0].astype(np.float64), K, V, 1.0 / math.sqrt(D))
        np.testing.assert_allclose(res[0], want, rtol=1e-12, atol=1e-12, err_msg=f"step {t}")
        if t == 0 and lag == 1:
            continue
        # the same step of a run INITIALISED with the longer history (static oracle: the partial chunk is an ordinary
        # candidate there, R22), with everything recalled at once
        n = len(flat)
        nch = -(-n // C)
        cold = np.zeros((nch, 2, C, D), np.float32)
        for s in range(n):
            cold[s // C, 0, s % C], cold[s // C, 1, s % C] = flat[s]
        st = LsaOracle(dtype="f32", H=H, D=D, C=C, W=W, k=nch, tau=1, recall_lag=0, hot_pages=2 * nch, W_q=orc.W_q, cold_csa=[cold],
                       n_csa=[n], chunk_emb=[np.ones((nch, 4), np.float32)], hca_k=[np.stack([a for a, _ in hca])],
                       hca_v=[np.stack([b for _, b in hca])], win_k=[win_k.copy()], win_v=[win_v.copy()], w_len=[orc.w_len[0]],
                       w_head=[orc.w_head[0]], step0=[0])
        st.step_begin(h)
        res2, _ = st.step_end(q)
        np.testing.assert_allclose(res[0], res2[0], rtol=1e-12, atol=1e-12, err_msg=f"static run, step {t}")


def test_invariants_over_a_seeded_run():
    """Small workload with the paper's cadences scaled down: each CSA entry attended at most once, the tail always attended,
    an exported chunk's cold copy = the rows that were handed over, at most two tier chunks, a completed chunk that is recalled
    later is fetched from the cold pool (its page holds the handed-over rows)."""
    cfg = make_small_config("f32", B=2, L=[4096 + 24, 2432], C=16, W=24, k=3 + TIER_SLOTS, tau=4, steps=0,
                            hot_pages=16 + 2 * TIER_SLOTS, needle_period=10 ** 9)
    wl = LsaWorkload(cfg)
    gi = GrowthInputs(wl, steps=200, csa_every=1, hca_every=16, hot_frac=1.0)
    orc = make_growing_oracle(wl, gi)
    assert orc.tier(0) == [cfg.n_csa(0) // cfg.C] and orc.tier(1) == []           # seq 0 starts with a partial chunk
    handed = {b: {} for b in range(cfg.B)}                                       # entry index -> (K row, V row)
    recalled_after_export = 0
    for t in range(200):
        n_before = list(orc.n_csa)
        done = oracle_appends(orc, gi, t)
        if gi.csa_due(t):
            e = gi.csa_entry(t)
            for b in range(cfg.B):
                handed[b][n_before[b]] = (e[0][b], e[1][b])
        for b, c in done:
            for i in range(cfg.C):
                s = c * cfg.C + i
                if s in handed[b]:
                    assert np.array_equal(orc.cold[b][c][0, i], handed[b][s][0]) and np.array_equal(orc.cold[b][c][1, i], handed[b][s][1])
        fired = orc.step_begin(wl.h(t))
        for b in range(cfg.B):
            tbl = orc.table(b)
            chunks = [c for c, _ in tbl]
            assert len(set(chunks)) == len(chunks) and chunks == sorted(chunks)
            assert len(orc.tier(b)) <= TIER_SLOTS and len(tbl) <= cfg.k
            if orc.n_csa[b] % cfg.C:
                assert chunks[-1] == orc.n_csa[b] // cfg.C                       # the tail is attended (P:185 tier 3)
            for c, p in orc.pool.cur[b]:
                assert p < orc.P_lru and np.array_equal(orc.pool.hot[p], orc.cold[b][c])
                if c >= cfg.n_chunks(b):                                         # a chunk completed during decode, recalled again
                    recalled_after_export += 1
        orc.step_end(wl.q(t), *wl.kv_new(t), attend=(t % 37 == 0))
    assert recalled_after_export > 0
    assert orc.exported == sum((orc.n_csa[b] // cfg.C) - (cfg.n_csa(b) // cfg.C) for b in range(cfg.B))
    assert orc.n_hca == [cfg.n_hca(b) + (199 // 16) for b in range(cfg.B)]


def test_without_appends_it_is_the_static_oracle_with_k_minus_2():
    cfg = make_small_config("f32", k=3 + TIER_SLOTS, hot_pages=16 + 2 * TIER_SLOTS, needle_period=10 ** 9)
    wl = LsaWorkload(cfg)
    gi = GrowthInputs(wl, steps=16)
    grow = make_growing_oracle(wl, gi)
    from lsa_harness import make_oracle
    stat = make_oracle(wl, k=3, hot_pages=16)
    for t in range(12):
        h, q = wl.h(t), wl.q(t)
        kn, vn = wl.kv_new(t)
        f1, f2 = grow.step_begin(h), stat.step_begin(h)
        assert sorted(f1) == sorted(f2)
        for b in f1:
            assert list(f1[b][0][:3]) == list(f2[b][0]) and f1[b][2] == f2[b][2]
        r1, r2 = grow.step_end(q, kn, vn), stat.step_end(q, kn, vn)
        np.testing.assert_array_equal(r1[0], r2[0])
        for b in range(cfg.B):
            assert grow.table(b) == stat.pool.cur[b]
