"""Parity of Level 2 (lsa_l2_init / lsa_l2_select / lsa_step_l2; Eq.(6)) against oracle/l2_oracle.py
on the same seeded inputs, through the C ABI, on the flagship shape (bf16, H=64, D=512, C=128: tcgen05 path).

Scores: the GPU multiplies bf16 inputs exactly and accumulates in fp32 (128 products per head, 64 heads), the oracle in
fp64: compared at rtol 1e-4 of the largest score.  Selection: a float decides an integer, so the entry SET must be the
oracle's except for swaps among entries whose oracle score lies within 1e-5 (relative) of the k2-th score
(BASELINE.json's rule for top-k); when the sets are identical - the normal case - the attention output is compared with
the oracle's own Level-2 attention at the BASELINE tolerance."""
import numpy as np
import pytest
import torch

from lsa_harness import GpuRig, attn_tolerance, make_oracle
from oracle import validate_selection
from oracle.l2_oracle import l2_decode_attention, l2_select, validate_l2_selection
from paper_2606_09079_b200.workloads import L2Inputs, LsaWorkload, make_config, make_small_config, to_torch

pytestmark = pytest.mark.gpu


def _rig(k, k2, B=2, L=(20096, 4992), steps=8, tau=4, dup_rows=0, **over):
    cfg = make_config(2, B=B, L=list(L), W=1024, k=k, tau=tau, steps=steps, q_gain=16.0,
                      hot_pages=2 * sum(min(k, -(-(l // 4) // 128)) for l in L) + 4, name="l2_parity", **over)
    wl = LsaWorkload(cfg)
    l2 = L2Inputs(wl)
    if dup_rows:                                              # only `dup_rows` distinct index keys per sequence: exact score ties
        l2.index_k = [K[np.arange(len(K)) % dup_rows].copy() for K in l2.index_k]
    rig = GpuRig(wl)
    rig.ctx.l2_init([to_torch(K, "bf16").to(rig.device) for K in l2.index_k], k2)
    return cfg, wl, l2, rig


def _dev_l2(rig, l2, t):
    return to_torch(l2.q_idx(t), "bf16").to(rig.device), torch.from_numpy(l2.w_idx(t)).to(rig.device)


def _forced(rig, orc, cfg, h, firing):
    forced = {}
    for b in firing:
        chunks, _ = rig.ctx.page_table(b, 0 if cfg.recall_lag == 0 else 1)
        sc = orc.scores(b, h[b])
        order = sorted(chunks, key=lambda ch: (-sc[ch], ch))
        padded = np.full(cfg.k, -1, dtype=np.int64); padded[: len(order)] = order
        assert validate_selection(padded, sc, cfg.k) is None
        forced[b] = chunks
    return forced


def _oracle_l2(orc, cfg, l2, t, k2):
    sels, ids, scs = [], [], []
    for b in range(cfg.B):
        s, i, sc = l2_select(l2.q_idx(t)[b], l2.w_idx(t)[b], l2.index_k[b], [c for c, _ in orc.pool.cur[b]], cfg.n_csa(b), cfg.C, k2)
        sels.append(s); ids.append(i); scs.append(sc)
    return sels, ids, scs


def _mask_of(cfg, orc, b, entries):
    m = np.zeros((cfg.k, cfg.C), dtype=bool)
    slot = {c: j for j, (c, _) in enumerate(orc.pool.cur[b])}          # tables are in ascending chunk id
    for s in entries:
        m[slot[int(s) // cfg.C], int(s) % cfg.C] = True
    return m


@pytest.mark.parametrize("k,k2,L", [(12, 37, (20096, 4992)), (12, 1, (20096, 4992)), (40, 700, (20096, 4992)), (40, 4096, (20096, 4992)),
                                    (72, 1500, (40960, 4992))])
def test_l2_select_and_attention_match_oracle(k, k2, L):
    """API level: lsa_l2_select then lsa_decode_attention.  k = 12: 1536 + 1248 entries (sort-all path); k = 40: 5024
    entries in sequence 0 (radix-select path), whose last chunk is partial (32 valid rows); k2 = 4096 covers all of
    sequence 1 (1248 entries): every valid row selected.  k2 = 1 / 37 leave most pages without a selected row."""
    cfg, wl, l2, rig = _rig(k, k2, L=L)
    orc = make_oracle(wl)
    tol = attn_tolerance("bf16")
    compared = 0
    for t in range(3):                                        # step 0 triggers, the table is current from step 1 on
        q, h = wl.q(t), wl.h(t)
        kn, vn = wl.kv_new(t)
        firing = [b for b in range(cfg.B) if orc.step[b] % cfg.tau == 0]
        rig.ctx.step(rig.dev(q), rig.dev(h), rig.dev(kn), rig.dev(vn))
        orc.step_begin(h, forced_selection=_forced(rig, orc, cfg, h, firing) if firing else None)
        orc.step_end(q, kn, vn, attend=False)
    for t in (3, 5):
        # the staged table of step 0 is current by now on both sides; no step counter moves below
        for b in range(cfg.B):
            orc.pool.maybe_swap(b, orc.step[b])
        qi, wi = _dev_l2(rig, l2, t)
        q = wl.q(t)
        sel, sc = rig.ctx.l2_select(qi, wi)
        out = rig.ctx.decode_attention(rig.dev(q))
        out_plain = rig.ctx.decode_attention(rig.dev(q))      # the selection is one-shot
        rig.ctx.sync()
        masks = [rig.ctx.l2_mask(b) for b in range(cfg.B)]    # written by the general (sorting) kernel
        rig.ctx.l2_select(qi, wi, want_entries=False)         # mask-only fast kernel (keys in registers, radix select)
        out_fast = rig.ctx.decode_attention(rig.dev(q))
        for b in range(cfg.B):
            assert np.array_equal(rig.ctx.l2_mask(b), masks[b]), f"t {t} seq {b}: the two Top-k kernels disagree"
            assert np.array_equal(masks[b], _mask_of(cfg, orc, b, [e for e in sel[b].cpu().tolist() if e >= 0]))
        assert torch.equal(out_fast, out)
        sel, sc = sel.cpu().numpy(), sc.cpu().numpy().astype(np.float64)
        o_sels, o_ids, o_scs = _oracle_l2(orc, cfg, l2, t, k2)
        same = True
        for b in range(cfg.B):
            assert len(o_ids[b]) == sum(orc.valid_rows(b, c) for c, _ in orc.pool.cur[b]) > 0
            msg = validate_l2_selection(sel[b], o_ids[b], o_scs[b], k2)
            assert msg is None, f"t {t} seq {b}: {msg}"
            n = min(k2, len(o_ids[b]))
            assert np.all(sel[b][n:] == -1) and np.all(sc[b][n:] == -np.inf)
            by_id = dict(zip(o_ids[b].tolist(), o_scs[b].tolist()))
            ref = np.array([by_id[int(e)] for e in sel[b][:n]])
            np.testing.assert_allclose(sc[b][:n], ref, rtol=0, atol=1e-4 * np.abs(o_scs[b]).max())
            assert np.all(sc[b][:n][:-1] >= sc[b][:n][1:]), "scores must come out in non-increasing order"
            same &= set(sel[b][:n].tolist()) == set(o_sels[b].tolist())
            if same and np.all(np.diff(np.sort(o_scs[b])) > 1e-5 * np.abs(o_scs[b]).max()):   # no near-ties: the ORDER is fixed too
                assert sel[b][:n].tolist() == o_sels[b].tolist()
        if same:
            ref_out, _ = l2_decode_attention(orc, q, o_sels)
            np.testing.assert_allclose(rig.host(out), ref_out, err_msg=f"Level-2 attention mismatch at t {t}", **tol)
            compared += 1
        ref_plain, _ = orc.decode_attention(q)
        np.testing.assert_allclose(rig.host(out_plain), ref_plain, **tol)
        if all(k2 >= len(o_ids[b]) for b in range(cfg.B)):
            assert torch.equal(out, out_plain)                # every valid row marked: the same arithmetic, bit for bit
    assert compared >= 1
    rig.ctx.close()


@pytest.mark.parametrize("k,k2", [(12, 300), (40, 1000)])
def test_l2_duplicate_keys_exact_ties_at_the_cutoff(k, k2):
    """Only 97 distinct index keys per sequence: the native scores come in groups of exactly equal values (identical
    inputs, identical arithmetic - on the GPU and in the oracle alike), and the k2-th score falls inside such a group, so
    the deterministic tie-break (score desc, entry id asc; M2) decides which members are kept.  Both Top-k kernels must
    return exactly the oracle's list."""
    cfg, wl, l2, rig = _rig(k, k2, dup_rows=97)
    orc = make_oracle(wl)
    for t in range(2):
        q, h = wl.q(t), wl.h(t)
        kn, vn = wl.kv_new(t)
        firing = [b for b in range(cfg.B) if orc.step[b] % cfg.tau == 0]
        rig.ctx.step(rig.dev(q), rig.dev(h), rig.dev(kn), rig.dev(vn))
        orc.step_begin(h, forced_selection=_forced(rig, orc, cfg, h, firing) if firing else None)
        orc.step_end(q, kn, vn, attend=False)
    for b in range(cfg.B):
        orc.pool.maybe_swap(b, orc.step[b])
    qi, wi = _dev_l2(rig, l2, 2)
    sel, sc = rig.ctx.l2_select(qi, wi)
    out = rig.ctx.decode_attention(rig.dev(wl.q(2)))
    masks = [rig.ctx.l2_mask(b) for b in range(cfg.B)]
    rig.ctx.l2_select(qi, wi, want_entries=False)
    out_fast = rig.ctx.decode_attention(rig.dev(wl.q(2)))
    rig.ctx.sync()
    o_sels, o_ids, o_scs = _oracle_l2(orc, cfg, l2, 2, k2)
    for b in range(cfg.B):
        n = min(k2, len(o_ids[b]))
        by_id = dict(zip(o_ids[b].tolist(), o_scs[b].tolist()))
        got = sel[b].cpu().numpy()
        # identical index-key rows must give identical oracle scores (same BLAS path for every row); if a host BLAS
        # ever rounded them differently the oracle's order inside a group would be arbitrary: fall back to the band rule
        groups_exact = all(len({by_id[e] for e in o_ids[b].tolist() if e % 97 == r}) <= 1 for r in range(97))
        if not groups_exact:
            assert validate_l2_selection(got, o_ids[b], o_scs[b], k2) is None
            continue
        if n < len(o_ids[b]):
            ranked = sorted(by_id, key=lambda e: (-by_id[e], e))
            assert by_id[ranked[n - 1]] == by_id[ranked[n]], "the cut-off must fall inside a tie group for this test to bite"
        assert got[:n].tolist() == o_sels[b].tolist(), f"seq {b}"
        assert np.array_equal(masks[b], _mask_of(cfg, orc, b, o_sels[b])) and np.array_equal(rig.ctx.l2_mask(b), masks[b])
    assert torch.equal(out, out_fast)
    ref, _ = l2_decode_attention(orc, wl.q(2), o_sels)
    np.testing.assert_allclose(rig.host(out), ref, **attn_tolerance("bf16"))
    rig.ctx.close()


def test_l2_all_scores_tied_selects_lowest_entry_ids():
    """Degenerate case: zero head weights make every native score exactly 0, so Eq.(6) is decided by the tie rule alone
    (M2): the k2 lowest entry ids of the resident set.  All 5024 keys of sequence 0 share one radix bin - more than the
    mask-only kernel's shared-memory candidate buffer holds - so its register fallback runs; both kernels must agree."""
    k2 = 700
    cfg, wl, l2, rig = _rig(40, k2)
    orc = make_oracle(wl)
    for t in range(2):
        q, h = wl.q(t), wl.h(t)
        kn, vn = wl.kv_new(t)
        firing = [b for b in range(cfg.B) if orc.step[b] % cfg.tau == 0]
        rig.ctx.step(rig.dev(q), rig.dev(h), rig.dev(kn), rig.dev(vn))
        orc.step_begin(h, forced_selection=_forced(rig, orc, cfg, h, firing) if firing else None)
        orc.step_end(q, kn, vn, attend=False)
    for b in range(cfg.B):
        orc.pool.maybe_swap(b, orc.step[b])
    qi, _ = _dev_l2(rig, l2, 2)
    wi = torch.zeros((cfg.B, 64), dtype=torch.float32, device=rig.device)
    sel, sc = rig.ctx.l2_select(qi, wi)
    out = rig.ctx.decode_attention(rig.dev(wl.q(2)))
    masks = [rig.ctx.l2_mask(b) for b in range(cfg.B)]
    rig.ctx.l2_select(qi, wi, want_entries=False)
    out_fast = rig.ctx.decode_attention(rig.dev(wl.q(2)))
    rig.ctx.sync()
    o_sels = []
    for b in range(cfg.B):
        o_sel, ids, o_sc = l2_select(l2.q_idx(2)[b], np.zeros(64, dtype=np.float32), l2.index_k[b], [c for c, _ in orc.pool.cur[b]],
                                     cfg.n_csa(b), cfg.C, k2)
        assert np.all(o_sc == 0.0) and o_sel.tolist() == ids[:k2].tolist()          # the oracle's own tie rule
        got = sel[b].cpu().numpy()
        assert got[got >= 0].tolist() == o_sel.tolist()                             # exact ties: the order is fixed too
        assert torch.all(sc[b][: len(o_sel)] == 0.0)
        assert np.array_equal(rig.ctx.l2_mask(b), masks[b]) and np.array_equal(masks[b], _mask_of(cfg, orc, b, o_sel))
        o_sels.append(o_sel)
    assert torch.equal(out, out_fast)
    ref, _ = l2_decode_attention(orc, wl.q(2), o_sels)
    np.testing.assert_allclose(rig.host(out), ref, **attn_tolerance("bf16"))
    rig.ctx.close()


def test_l2_before_any_trigger_attends_hca_and_window_only():
    cfg, wl, l2, rig = _rig(12, 64)
    orc = make_oracle(wl)
    qi, wi = _dev_l2(rig, l2, 0)
    q = wl.q(0)
    sel, sc = rig.ctx.l2_select(qi, wi)                       # empty tables: nothing to select
    out = rig.ctx.decode_attention(rig.dev(q))
    rig.ctx.l2_select(qi, wi, want_entries=False)
    assert not rig.ctx.l2_mask(0).any() and not rig.ctx.l2_mask(1).any()
    assert torch.equal(rig.ctx.decode_attention(rig.dev(q)), out)
    rig.ctx.sync()
    assert torch.all(sel == -1) and torch.all(sc == -float("inf"))
    ref, _ = l2_decode_attention(orc, q, [[] for _ in range(cfg.B)])
    np.testing.assert_allclose(rig.host(out), ref, **attn_tolerance("bf16"))
    rig.ctx.close()


@pytest.mark.parametrize("recall_lag", [1, 0])
def test_lsa_step_l2_lockstep(recall_lag):
    """lsa_step_l2 over several trigger periods: Level 1 (dual encoder) recalls pages, Level 2 picks k2 entries of the
    current tables every step, attention runs over HCA (+) those (+) the growing window; outputs vs the oracle."""
    k2 = 200
    cfg, wl, l2, rig = _rig(12, k2, steps=10, tau=4, recall_lag=recall_lag)
    orc = make_oracle(wl)
    tol = attn_tolerance("bf16")
    max_err = 0.0
    for t in range(cfg.steps):
        q, h = wl.q(t), wl.h(t)
        kn, vn = wl.kv_new(t)
        qi, wi = _dev_l2(rig, l2, t)
        firing = [b for b in range(cfg.B) if orc.step[b] % cfg.tau == 0]
        out = rig.ctx.step_l2(rig.dev(q), rig.dev(h), rig.dev(kn), rig.dev(vn), qi, wi)
        orc.step_begin(h, forced_selection=_forced(rig, orc, cfg, h, firing) if firing else None)
        o_sels, o_ids, o_scs = _oracle_l2(orc, cfg, l2, t, k2)
        if t == 0 and recall_lag == 1:
            assert all(len(i) == 0 for i in o_ids)            # the first recall is visible one step later
        orc.step_end(q, kn, vn, attend=False)                 # (d) append, (f) counters; (e) is Level-2 attention:
        orc_step = list(orc.step)
        ref, _ = l2_decode_attention(orc, q, o_sels)
        got = rig.host(out)
        np.testing.assert_allclose(got, ref, err_msg=f"step {t}", **tol)
        max_err = max(max_err, float(np.abs(got - ref).max()))
        assert orc.step == orc_step
    # Level 2 changes the result: the same step without it differs from the Level-2 output
    plain = rig.host(rig.ctx.decode_attention(rig.dev(q)))
    assert np.abs(plain - got).max() > 10 * max(max_err, 1e-4)
    rig.ctx.close()


def test_l2_cfg3_full_size_bench_launch_config():
    """BASELINE config 3 (1M context, k = 64 -> 8192 resident entries) with k2 = 2048, the configuration `bench.py --l2`
    times: trigger step, the step whose table swap rides on the masked attention launch, and a plain step."""
    cfg = make_config(3)
    wl = LsaWorkload(cfg)
    l2 = L2Inputs(wl)
    rig = GpuRig(wl)
    k2 = 2048
    rig.ctx.l2_init([to_torch(K, "bf16").to(rig.device) for K in l2.index_k], k2)
    orc = make_oracle(wl)
    tol = attn_tolerance("bf16")
    for t in range(3):
        q, h = wl.q(t), wl.h(t)
        kn, vn = wl.kv_new(t)
        qi, wi = _dev_l2(rig, l2, t)
        firing = [b for b in range(cfg.B) if orc.step[b] % cfg.tau == 0]
        out = rig.ctx.step_l2(rig.dev(q), rig.dev(h), rig.dev(kn), rig.dev(vn), qi, wi)
        orc.step_begin(h, forced_selection=_forced(rig, orc, cfg, h, firing) if firing else None)
        o_sels, o_ids, o_scs = _oracle_l2(orc, cfg, l2, t, k2)
        orc.step_end(q, kn, vn, attend=False)
        if t > 0:
            assert len(o_ids[0]) == 8192 and len(o_sels[0]) == k2
            mask = rig.ctx.l2_mask(0)
            assert mask.sum() == k2
            got_set = {int(orc.pool.cur[0][j][0]) * cfg.C + int(r) for j, r in zip(*np.nonzero(mask))}
            padded = np.full(k2, -1, dtype=np.int64); padded[:] = sorted(got_set)
            assert validate_l2_selection(padded, o_ids[0], o_scs[0], k2) is None
            if got_set != set(o_sels[0].tolist()):
                continue                                              # a near-tie at the cut-off went the other way
        ref, _ = l2_decode_attention(orc, q, o_sels)
        np.testing.assert_allclose(rig.host(out), ref, err_msg=f"step {t}", **tol)
    rig.ctx.close()


def test_l2_rejects_unsupported():
    from paper_2606_09079_b200 import lsa
    cfg = make_small_config("bf16", B=1, L=[4096], C=16, H=8, D=64, Dh=128, E=64, k=3, hot_pages=16, W=64)
    rig = GpuRig(LsaWorkload(cfg))
    z = torch.zeros((1024, 128), dtype=torch.bfloat16, device=rig.device)
    with pytest.raises(lsa.LsaError) as e:
        rig.ctx.l2_init([z], 16)                               # SIMT shape: no Level-2 kernel
    assert e.value.code == -6
    with pytest.raises(lsa.LsaError):
        rig.ctx.step_l2(z, z, None, None, z, z.float())        # not initialised
    rig.ctx.close()
    cfg2, wl2, l22, rig2 = _rig(12, 8)
    with pytest.raises(lsa.LsaError):
        rig2.ctx.l2_init([to_torch(K, "bf16").to(rig2.device) for K in l22.index_k], 8)   # twice
    rig2.ctx.close()
