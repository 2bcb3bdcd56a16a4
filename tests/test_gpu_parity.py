"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): chunk indices, page tables, residency, counters and fetched bytes
bit-exact (selection swaps only inside the 1e-5-relative band around the k-th oracle score, never
among bit-identical scores); attention within abs 2e-2 / rel 1e-2 (bf16) or 1e-4 (fp32).
"""
import math

import numpy as np
import pytest
import torch

from lsa_harness import GpuRig, attn_tolerance, make_oracle, run_lockstep
from oracle import ResidencyOracle, attention, chunk_scores, query_tower, topk_select, validate_selection, widen
from paper_2606_09079_b200.workloads import (LsaWorkload, as_f64, from_torch, make_config, make_small_config,
                                             plant_boundary_ties, store, to_torch)

pytestmark = pytest.mark.gpu


def _lsa():
    from paper_2606_09079_b200 import lsa
    return lsa


# ------------------------------------------------------------------------------- S1-S3
@pytest.mark.parametrize("n_fire", [1, 3, 8, 11, 16, 20])
def test_index_select_batched_tower_on_tensor_cores(n_fire):
    """S1 for 8..16 sequences firing together is one tcgen05 GEMM (lsa_index_tc.cu: W_q streamed once, the sequences on N,
    partial sums over slices of Dh added in a fixed order by the scoring kernel); fewer sequences, or a batch of 20 (16 + 4),
    take the GEMV.  Scores element by element and the selection against the oracle at the BASELINE shape Dh = 4096, E = 512;
    the 8 sequences of a batched call must also get exactly the chunks they get when they fire alone."""
    cfg = make_small_config("bf16", B=20, L=[4096 + 512 * b for b in range(20)], C=16, H=8, D=64, E=512, Dh=4096, k=12, hot_pages=600, W=64)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    h = wl.h(0)
    ids = list(range(n_fire))
    sel, sc = rig.ctx.index_select(rig.dev(h[:n_fire]), ids)
    rig.ctx.sync()
    sel, sc = sel.cpu().numpy(), sc.cpu().numpy().astype(np.float64)
    for i, b in enumerate(ids):
        ref = chunk_scores(query_tower(wl.W_q, h[b]), wl.chunk_emb(b, 0))
        assert validate_selection(sel[i], ref, cfg.k) is None
        np.testing.assert_allclose(sc[i][sel[i] >= 0], ref[sel[i][sel[i] >= 0]], atol=2e-6)
    if n_fire >= 8:
        for b in (0, n_fire - 1):
            alone, _ = rig.ctx.index_select(rig.dev(h[b:b + 1]), [b])
            rig.ctx.sync()
            assert np.array_equal(alone.cpu().numpy()[0], sel[b])
    rig.ctx.close()


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_index_select_matches_oracle_order(dtype):
    cfg = make_small_config(dtype, B=3, L=[65536, 32768, 1024], C=16, E=128, Dh=512, k=24, hot_pages=256)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    orc = make_oracle(wl)
    for t in (0, 5):
        h = wl.h(t)
        sel, sc = rig.ctx.index_select(rig.dev(h), [0, 1, 2])
        rig.ctx.sync()
        sel, sc = sel.cpu().numpy(), sc.cpu().numpy().astype(np.float64)
        for b in range(cfg.B):
            osc = orc.scores(b, h[b])
            assert validate_selection(sel[b], osc, cfg.k) is None
            ke = cfg.k_eff(b)
            np.testing.assert_allclose(sc[b, :ke], osc[sel[b, :ke]], atol=2e-6, rtol=1e-5)
            assert np.all(sc[b, ke:] == -np.inf)
    # subset call: rows of h follow seq_ids
    h = wl.h(9)
    sel2, _ = rig.ctx.index_select(rig.dev(h[[2, 0]][::-1].copy()), [0, 2])
    sel_all, _ = rig.ctx.index_select(rig.dev(h), [0, 1, 2])
    rig.ctx.sync()
    assert torch.equal(sel2[0], sel_all[0]) and torch.equal(sel2[1], sel_all[2])


def test_index_select_exact_ties_and_zero_query():
    cfg = make_config(5, B=2, L=[524288, 524288], hot_pages=512)
    wl = LsaWorkload(cfg, build_kv=False)
    # index-only context: K/V tensors are tiny dummies
    lsa = _lsa()
    dev = torch.device("cuda:0")
    orc_scores = []
    embs = []
    h = wl.h(0)
    for b in range(cfg.B):
        emb = wl.chunk_emb(b, 0)
        qh = query_tower(wl.W_q, h[b])
        order = topk_select(chunk_scores(qh, emb), cfg.n_chunks(b))[0]
        emb = plant_boundary_ties(emb, order, cfg.k, cfg.dtype)
        if b == 1:            # many exact duplicates of the best row
            emb[100:140] = emb[order[0]]
        embs.append(emb)
        orc_scores.append(chunk_scores(qh, emb))
    cold = [torch.zeros((cfg.n_chunks(b), 2, cfg.C, cfg.D), dtype=torch.bfloat16).pin_memory() for b in range(cfg.B)]
    emb_d = [to_torch(e, "bf16").to(dev) for e in embs]
    z = torch.zeros((8, cfg.D), dtype=torch.bfloat16, device=dev)
    seqs = [dict(cold_csa=cold[b], n_csa=cfg.n_csa(b), chunk_emb=emb_d[b], hca_k=z, hca_v=z, win_k=z.clone(),
                 win_v=z.clone(), w_len=0) for b in range(cfg.B)]
    ctx = lsa.LsaContext(dtype=lsa.LSA_BF16, H=cfg.H, D=cfg.D, C_=cfg.C, W=8, Dh=cfg.Dh, E=cfg.E, k=cfg.k, tau=cfg.tau,
                         hot_pool=torch.zeros((cfg.hot_pages, 2, cfg.C, cfg.D), dtype=torch.bfloat16, device=dev),
                         W_q=to_torch(wl.W_q, "bf16").to(dev), seqs=seqs)
    sel, sc = ctx.index_select(to_torch(h, "bf16").to(dev), [0, 1])
    ctx.sync()
    sel = sel.cpu().numpy()
    for b in range(cfg.B):
        assert validate_selection(sel[b], orc_scores[b], cfg.k) is None
    dup = set(range(100, 140))
    got = [c for c in sel[1].tolist() if c in dup or orc_scores[1][c] == orc_scores[1][100]]
    assert got == sorted(got)                          # equal scores come out in ascending chunk id
    # zero hidden state: every score is 0 -> lowest chunk ids (R16)
    sel0, sc0 = ctx.index_select(torch.zeros((2, cfg.Dh), dtype=torch.bfloat16, device=dev), [0, 1])
    ctx.sync()
    assert sel0[0].tolist() == list(range(cfg.k)) and torch.all(sc0 == 0)
    ctx.close()


def test_topk_radix_path_many_chunks():
    """n_chunks > 4096 exercises the radix-select branch of S3."""
    cfg = make_small_config("f32", B=1, L=[6000 * 16 * 4], C=16, D=64, H=8, E=64, Dh=128, k=50, hot_pages=128,
                            emb_mode="uniform", n_needles=0)
    wl = LsaWorkload(cfg)
    assert cfg.n_chunks(0) == 6000
    rig = GpuRig(wl)
    orc = make_oracle(wl)
    for t in range(3):
        h = wl.h(t)
        sel, sc = rig.ctx.index_select(rig.dev(h), [0])
        rig.ctx.sync()
        assert validate_selection(sel[0].cpu().numpy(), orc.scores(0, h[0]), cfg.k) is None


# ------------------------------------------------------------------------------- S4-S5
@pytest.mark.parametrize("lag", [0, 1])
def test_fetch_chunks_lockstep_random_selections(lag):
    cfg = make_small_config("bf16", B=3, L=[4096, 2432, 1280], C=16, k=5, hot_pages=30 + 3, recall_lag=lag)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    n_chunks = [cfg.n_chunks(b) for b in range(cfg.B)]
    ref = ResidencyOracle(cfg.B, n_chunks, cfg.hot_pages, wl.cold_csa)
    g = np.random.default_rng(5)
    for it in range(25):
        ids = sorted(g.choice(cfg.B, size=g.integers(1, cfg.B + 1), replace=False).tolist())
        sel = np.full((len(ids), cfg.k), -1, dtype=np.int32)
        for i, b in enumerate(ids):
            ke = min(cfg.k, n_chunks[b])
            sel[i, :ke] = g.choice(n_chunks[b], size=ke, replace=False)
        rig.ctx.fetch_chunks(ids, torch.from_numpy(sel).to(rig.device))
        for i, b in enumerate(ids):
            ref.fetch(b, sel[i], 0, 0)
        for b in ids:
            ch, pg = rig.ctx.page_table(b, 1)
            assert list(zip(ch, pg)) == ref.nxt[b]
        rig.ctx.commit_tables()
        for b in range(cfg.B):
            ref.maybe_swap(b, 0)
            ch, pg = rig.ctx.page_table(b, 0)
            assert list(zip(ch, pg)) == ref.cur[b]
            assert rig.ctx.residency(b, n_chunks[b]) == ref.page_of[b]
        st = rig.ctx.stats()
        assert (st["hits"], st["misses"], st["evictions"], st["bytes_fetched"]) == \
               (ref.hits, ref.misses, ref.evictions, ref.bytes_fetched)
        hot = from_torch(rig.hot_pool.cpu(), "bf16")
        owned = [p for p, o in enumerate(ref.owner) if o is not None]
        assert np.array_equal(hot[owned], ref.hot[owned])
    assert ref.evictions > 0


def test_residency_radix_path_many_pages():
    """hot_pages > 4096 exercises the radix-select branch of S4 (victim selection)."""
    cfg = make_small_config("f32", B=2, L=[6000 * 16 * 4, 3000 * 16 * 4], C=16, D=64, H=8, E=64, Dh=128, k=40,
                            hot_pages=5000, emb_mode="uniform", n_needles=0, recall_lag=0)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    n_chunks = [cfg.n_chunks(b) for b in range(cfg.B)]
    ref = ResidencyOracle(cfg.B, n_chunks, cfg.hot_pages, wl.cold_csa)
    g = np.random.default_rng(6)
    for it in range(140):                              # 140 * 80 selections > 5000 pages -> LRU kicks in
        sel = np.stack([g.choice(n_chunks[b], size=cfg.k, replace=False) for b in range(2)]).astype(np.int32)
        rig.ctx.fetch_chunks([0, 1], torch.from_numpy(sel).to(rig.device))
        rig.ctx.commit_tables()
        for b in range(2):
            ref.fetch(b, sel[b], 0, 0)
            ref.maybe_swap(b, 0)
        if it % 20 == 19 or it > 130:
            for b in range(2):
                ch, pg = rig.ctx.page_table(b, 0)
                assert list(zip(ch, pg)) == ref.cur[b], f"iteration {it}"
    st = rig.ctx.stats()
    assert ref.evictions > 0 and (st["hits"], st["misses"], st["evictions"]) == (ref.hits, ref.misses, ref.evictions)


def test_init_rejects_unpinned_and_small_pool():
    lsa = _lsa()
    cfg = make_small_config("f32")
    wl = LsaWorkload(cfg)
    with pytest.raises(lsa.LsaError, match="hot_pages"):
        GpuRig(LsaWorkload(make_small_config("f32", hot_pages=5)))
    rig = GpuRig(wl)
    z = torch.zeros((4, cfg.D), device=rig.device)
    with pytest.raises(lsa.LsaError, match="pinned"):
        lsa.LsaContext(dtype=0, H=cfg.H, D=cfg.D, C_=cfg.C, W=4, Dh=cfg.Dh, E=cfg.E, k=1, tau=4, hot_pool=rig.hot_pool,
                       W_q=rig.W_q, seqs=[dict(cold_csa=torch.zeros((2, 2, cfg.C, cfg.D)), n_csa=20, chunk_emb=rig.emb[0],
                                               hca_k=z, hca_v=z, win_k=z.clone(), win_v=z.clone())])
    with pytest.raises(lsa.LsaError, match="UNSUPPORTED"):
        lsa.LsaContext(dtype=0, H=24, D=64, C_=cfg.C, W=4, Dh=cfg.Dh, E=cfg.E, k=1, tau=4, hot_pool=rig.hot_pool,
                       W_q=rig.W_q, seqs=[dict(cold_csa=rig.cold[0], n_csa=20, chunk_emb=rig.emb[0], hca_k=z, hca_v=z,
                                               win_k=z.clone(), win_v=z.clone())])


# ------------------------------------------------------------------------------- S7-S8
def _direct_ctx(dtype, H, D, C, hca_k, hca_v, win_k, win_v, w_len, W, **kw):
    """A context with no CSA chunks at all: attention over HCA + window only."""
    lsa = _lsa()
    dev = torch.device("cuda:0")
    tdt = torch.float32 if dtype == "f32" else torch.bfloat16
    B = len(hca_k)
    seqs = [dict(cold_csa=None, n_csa=0, chunk_emb=None, hca_k=hca_k[b], hca_v=hca_v[b], win_k=win_k[b], win_v=win_v[b],
                 w_len=w_len[b]) for b in range(B)]
    return lsa.LsaContext(dtype=0 if dtype == "f32" else 1, H=H, D=D, C_=C, W=W, Dh=64, E=64, k=1, tau=4,
                          hot_pool=torch.zeros((2 * B, 2, C, D), dtype=tdt, device=dev),
                          W_q=torch.zeros((64, 64), dtype=tdt, device=dev), seqs=seqs, **kw)


@pytest.mark.parametrize("dtype,H,D", [("f32", 16, 128), ("bf16", 64, 512), ("bf16", 8, 64), ("f32", 64, 64)])
def test_attention_edge_cases(dtype, H, D):
    dev = torch.device("cuda:0")
    tdt = torch.float32 if dtype == "f32" else torch.bfloat16
    g = torch.Generator().manual_seed(1)
    W = 40
    rnd = lambda *s: (torch.randn(*s, generator=g)).to(tdt).to(dev)
    # seq 0: exactly one key (in HCA), empty window; seq 1: no keys at all; seq 2: all keys equal;
    # seq 3: ragged 37 HCA rows + 29 window rows with large logits
    hk = [rnd(1, D), torch.zeros((0, D), dtype=tdt, device=dev), rnd(1, D).expand(33, D).contiguous(), rnd(37, D)]
    hv = [rnd(1, D), torch.zeros((0, D), dtype=tdt, device=dev), rnd(33, D), rnd(37, D)]
    wk = [rnd(W, D) for _ in range(4)]
    wv = [rnd(W, D) for _ in range(4)]
    w_len = [0, 0, 0, 29]
    ctx = _direct_ctx(dtype, H, D, 16, hk, hv, wk, wv, w_len, W, sm_scale=0.5)
    q = rnd(4, H, D)
    out, lse = ctx.decode_attention(q, want_lse=True)
    ctx.sync()
    out64 = out.double().cpu().numpy()
    lse = lse.cpu().numpy()
    tol = attn_tolerance(dtype)
    # single key -> exactly that key's value
    assert torch.equal(out[0], hv[0].expand(H, D)), "single-key attention must return the value row bit-exactly"
    # no keys -> zeros, lse = -inf
    assert torch.all(out[1] == 0) and np.all(lse[1] == -np.inf)
    # equal keys -> mean of V
    np.testing.assert_allclose(out64[2], np.broadcast_to(hv[2].double().mean(0).cpu().numpy(), (H, D)), **tol)
    # ragged + large logits vs oracle
    K = np.concatenate([hk[3].double().cpu().numpy(), wk[3][:29].double().cpu().numpy()])
    V = np.concatenate([hv[3].double().cpu().numpy(), wv[3][:29].double().cpu().numpy()])
    ref, ref_lse, _ = attention(q[3].double().cpu().numpy(), K, V, 0.5)
    np.testing.assert_allclose(out64[3], ref, **tol)
    np.testing.assert_allclose(lse[3], ref_lse, atol=2e-2 if dtype == "bf16" else 1e-4, rtol=1e-3)
    ctx.close()


@pytest.mark.parametrize("merge", ["kernel", "fused"])
@pytest.mark.parametrize("keep", [(0, 1, 2, 3, 4), (0, 1, 2, 4), (4,)])
@pytest.mark.parametrize("max_ctas", [0, 1, 5])
def test_tcgen05_attention_edge_cases(max_ctas, keep, merge):
    """The tensor-core kernel (bf16, H=64, D=512, C=128): single key, no keys, equal keys, ragged
    segments, and a running maximum that jumps by far more than 2^8 between tiles (O rescale path).
    S8 as the separate combine kernel (two-phase for 5 sequences, single-round-trip for <= 4) and fused
    behind the attention kernel's grid barrier (<= 4 sequences; ignored for 5)."""
    lsa = _lsa()
    dev = torch.device("cuda:0")
    H, D, W = 64, 512, 200
    g = torch.Generator().manual_seed(2)
    rnd = lambda *s: torch.randn(*s, generator=g).to(torch.bfloat16).to(dev)
    qdir = torch.randn(D, generator=g)
    qdir = qdir / qdir.norm()
    ramp = (torch.arange(700).float()[:, None] / 700.0 * 90.0) * qdir[None, :]            # logits grow with the row id
    ramp_k = (ramp + 0.05 * torch.randn(700, D, generator=g)).to(torch.bfloat16).to(dev)
    hk = [rnd(1, D), torch.zeros((0, D), dtype=torch.bfloat16, device=dev), rnd(1, D).expand(333, D).contiguous(), rnd(37, D), ramp_k]
    hv = [rnd(1, D), torch.zeros((0, D), dtype=torch.bfloat16, device=dev), rnd(333, D), rnd(37, D), rnd(700, D)]
    wk = [rnd(W, D) for _ in range(5)]
    wv = [rnd(W, D) for _ in range(5)]
    w_len = [0, 0, 0, 29, 130]
    q = rnd(5, H, D)
    q[4] = (qdir[None, :] * (1.0 + 0.1 * torch.rand(H, 1, generator=g))).to(torch.bfloat16).to(dev)
    sel = lambda xs: [xs[i] for i in keep]
    hk, hv, wk, wv, w_len, q = sel(hk), sel(hv), sel(wk), sel(wv), sel(w_len), q[list(keep)].contiguous()
    ctx = _direct_ctx("bf16", H, D, 128, hk, hv, wk, wv, w_len, W, sm_scale=0.5, max_ctas=max_ctas,
                      attn_impl=lsa.LSA_ATTN_TCGEN05,
                      merge_mode=lsa.LSA_MERGE_FUSED if merge == "fused" else lsa.LSA_MERGE_KERNEL)
    assert ctx.stats()["attn_impl"] == lsa.LSA_ATTN_TCGEN05
    for rep in range(3):                      # repeated launches: the arrival counter of the fused merge keeps counting
        out, lse = ctx.decode_attention(q, want_lse=True)
    ctx.sync()
    out64, lse = out.double().cpu().numpy(), lse.cpu().numpy()
    tol = attn_tolerance("bf16")
    for i, orig in enumerate(keep):
        if orig == 0:
            assert torch.equal(out[i], hv[i].expand(H, D)), "single-key attention must return the value row bit-exactly"
        elif orig == 1:
            assert torch.all(out[i] == 0) and np.all(lse[i] == -np.inf)
        elif orig == 2:
            np.testing.assert_allclose(out64[i], np.broadcast_to(hv[i].double().mean(0).cpu().numpy(), (H, D)), **tol)
        else:
            K = np.concatenate([hk[i].double().cpu().numpy(), wk[i][: w_len[i]].double().cpu().numpy()])
            V = np.concatenate([hv[i].double().cpu().numpy(), wv[i][: w_len[i]].double().cpu().numpy()])
            ref, ref_lse, _ = attention(q[i].double().cpu().numpy(), K, V, 0.5)
            np.testing.assert_allclose(out64[i], ref, **tol)
            np.testing.assert_allclose(lse[i], ref_lse, atol=2e-2, rtol=1e-3)
    ctx.close()


@pytest.mark.parametrize("merge", ["kernel", "fused"])
@pytest.mark.parametrize("v_scale", [2.0 ** -40, 1.0, 2.0 ** 40])
def test_tcgen05_partials_keep_precision_at_any_magnitude(v_scale, merge):
    """The split-K partials are fp16 with a power-of-two scale per block (lsa_attn_tc_defs.cuh): values far
    outside fp16's own range (V ~ 2^-40 or 2^40) and a row whose columns differ by 2^20 must come out with the
    same RELATIVE accuracy as values near 1.  Several CTAs per sequence so the partials really are merged."""
    lsa = _lsa()
    dev = torch.device("cuda:0")
    H, D, W = 64, 512, 128
    g = torch.Generator().manual_seed(21)
    rnd = lambda *s: torch.randn(*s, generator=g)
    n_rows = [2000, 777]
    col_gain = torch.ones(D)
    col_gain[::7] = 2.0 ** 20                                     # wide dynamic range inside one row of V
    hk = [rnd(n, D).to(torch.bfloat16).to(dev) for n in n_rows]
    hv = [(rnd(n, D) * col_gain * v_scale).to(torch.bfloat16).to(dev) for n in n_rows]
    wk = [rnd(W, D).to(torch.bfloat16).to(dev) for _ in n_rows]
    wv = [(rnd(W, D) * col_gain * v_scale).to(torch.bfloat16).to(dev) for _ in n_rows]
    w_len = [100, 0]
    q = rnd(2, H, D).to(torch.bfloat16).to(dev)                   # logits ~ N(0, 5.6^2): a few keys dominate, |out| ~ |V|
    ctx = _direct_ctx("bf16", H, D, 128, hk, hv, wk, wv, w_len, W, sm_scale=0.25, attn_impl=lsa.LSA_ATTN_TCGEN05,
                      merge_mode=lsa.LSA_MERGE_FUSED if merge == "fused" else lsa.LSA_MERGE_KERNEL)
    out = ctx.decode_attention(q)
    ctx.sync()
    assert ctx.stats()["attn_ctas"] > 4
    out64 = out.double().cpu().numpy()
    for b in range(2):
        K = np.concatenate([hk[b].double().cpu().numpy(), wk[b][: w_len[b]].double().cpu().numpy()])
        V = np.concatenate([hv[b].double().cpu().numpy(), wv[b][: w_len[b]].double().cpu().numpy()])
        ref, _, _ = attention(q[b].double().cpu().numpy(), K, V, 0.25)
        gain = (col_gain.double() * v_scale).numpy()[None, :]
        assert np.abs(ref / gain).mean() > 0.1
        # relative to each column's magnitude, tighter than the north star's bf16 bar (abs 2e-2 / rel 1e-2)
        np.testing.assert_allclose(out64[b] / gain, ref / gain, atol=1e-2, rtol=1e-2)
    ctx.close()


@pytest.mark.parametrize("merge", ["kernel", "fused"])
def test_tcgen05_contexts_of_one_stream_share_the_workspace(merge):
    """Contexts on the same compute stream share the split-K workspace (lsa_attn_tc.cu): launches of three
    contexts with different batch sizes and key counts, interleaved back to back without a host sync, must each
    match the oracle - also after one of them was closed while the others keep running."""
    lsa = _lsa()
    dev = torch.device("cuda:0")
    H, D, W = 64, 512, 256
    g = torch.Generator().manual_seed(11)
    rnd = lambda *s: torch.randn(*s, generator=g).to(torch.bfloat16).to(dev)
    st = torch.cuda.Stream(dev)
    shapes = [[1500, 700], [3000], [130, 0, 900, 257, 64]]          # HCA rows per sequence, per context
    rigs = []
    for n_rows in shapes:
        B = len(n_rows)
        hk, hv = [rnd(n, D) for n in n_rows], [rnd(n, D) for n in n_rows]
        wk, wv = [rnd(W, D) for _ in range(B)], [rnd(W, D) for _ in range(B)]
        w_len = [(37 * (b + 1)) % W for b in range(B)]
        ctx = _direct_ctx("bf16", H, D, 128, hk, hv, wk, wv, w_len, W, sm_scale=0.05, attn_impl=lsa.LSA_ATTN_TCGEN05,
                          stream_compute=st, merge_mode=lsa.LSA_MERGE_FUSED if merge == "fused" else lsa.LSA_MERGE_KERNEL)
        rigs.append(dict(ctx=ctx, hk=hk, hv=hv, wk=wk, wv=wv, w_len=w_len, q=rnd(B, H, D),
                         out=torch.empty((B, H, D), dtype=torch.bfloat16, device=dev)))
    tol = attn_tolerance("bf16")
    torch.cuda.synchronize()

    def check(r):
        out64 = r["out"].double().cpu().numpy()
        for b in range(len(r["hk"])):
            K = np.concatenate([r["hk"][b].double().cpu().numpy(), r["wk"][b][: r["w_len"][b]].double().cpu().numpy()])
            V = np.concatenate([r["hv"][b].double().cpu().numpy(), r["wv"][b][: r["w_len"][b]].double().cpu().numpy()])
            ref, _, _ = attention(r["q"][b].double().cpu().numpy(), K, V, 0.05)
            np.testing.assert_allclose(out64[b], ref, **tol)

    for rep in range(4):
        for r in rigs:
            r["ctx"].decode_attention(r["q"], r["out"])
    st.synchronize()
    for r in rigs:
        check(r)
    rigs[0]["ctx"].close()                      # the first context created the workspace; the others keep it alive
    for rep in range(3):
        for r in rigs[1:]:
            with torch.cuda.stream(st):
                r["out"].zero_()
            r["ctx"].decode_attention(r["q"], r["out"])
    st.synchronize()
    for r in rigs[1:]:
        check(r)
        r["ctx"].close()


@pytest.mark.parametrize("impl", ["simt", "tcgen05", "tcgen05_merge_fused"])
def test_flagship_shape_short_context_both_impls(impl):
    """bf16 H=64 D=512 C=128 at a short context, with a partial last chunk, through both kernels; the
    tensor-core kernel with S8 fused behind its grid barrier (B <= 4 default) and as a separate kernel."""
    lsa = _lsa()
    cfg = make_config(2, L=[16384 + 4 * 37], W=1024, k=6, hot_pages=16, steps=70, name="cfg2_short", q_gain=16.0, tau=32)
    assert cfg.n_csa(0) % cfg.C != 0
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl, attn_impl=lsa.LSA_ATTN_SIMT if impl == "simt" else lsa.LSA_ATTN_TCGEN05,
                 merge_mode=lsa.LSA_MERGE_FUSED if impl.endswith("merge_fused") else lsa.LSA_MERGE_AUTO)
    r = run_lockstep(wl, rig, cfg.steps, check_attention_at={0, 1, 2, 31, 32, 33, 34, 64, 65, 69})
    assert r["checked"] == 10


@pytest.mark.parametrize("merge", ["kernel", "fused"])
def test_flagship_shape_growing_window_and_ring_wrap(merge):
    """S6 and the window append ride on the attention launch on steps without a trigger (tensor-core path).
    Growing ring: w_len starts at a multiple of 128, so the first appended token opens a new tile and later
    ones extend a ragged tile; full ring: w_head wraps and the oldest row is replaced.  Two sequences, so the
    appended rows land in tiles owned by different CTAs."""
    lsa = _lsa()
    mm = lsa.LSA_MERGE_FUSED if merge == "fused" else lsa.LSA_MERGE_KERNEL
    # (a) growing: L = 8576 = 67 * 128 < W
    cfg = make_config(2, B=2, L=[8576, 4096 + 4 * 30], W=9000, k=5, hot_pages=24, steps=12, name="cfg2_growing", q_gain=16.0, tau=4)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl, attn_impl=lsa.LSA_ATTN_TCGEN05, merge_mode=mm)
    r = run_lockstep(wl, rig, cfg.steps)
    assert r["checked"] == cfg.steps
    rig.ctx.close()
    # (b) full ring of 300 rows (not a multiple of 128): 310 steps wrap w_head once
    cfg = make_config(2, B=2, L=[16384, 8192], W=300, k=4, hot_pages=16, steps=310, name="cfg2_wrap", q_gain=16.0, tau=64)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl, attn_impl=lsa.LSA_ATTN_TCGEN05, merge_mode=mm)
    r = run_lockstep(wl, rig, cfg.steps, check_attention_at={0, 1, 2, 63, 64, 65, 127, 128, 129, 255, 256, 298, 299, 300, 301, 309})
    assert r["checked"] == 16
    rig.ctx.close()


@pytest.mark.parametrize("pinned_out", [True, False])
def test_step_host_equals_step(pinned_out):
    """lsa_step_host gives bit-identical outputs, page tables and counters to lsa_step, with pinned buffers
    (inputs pulled by a gather kernel, result written in place) and pageable ones (packed copy in, copy out)."""
    lsa = _lsa()
    cfg = make_config(2, B=2, L=[16384 + 4 * 37, 8192], W=1024, k=6, hot_pages=32, steps=40, name="cfg2_host", q_gain=16.0, tau=8)
    wl = LsaWorkload(cfg)
    a, b_ = GpuRig(wl), GpuRig(wl)
    out_h = torch.empty((cfg.B, cfg.H, cfg.D), dtype=torch.bfloat16)
    if pinned_out:
        out_h = out_h.pin_memory()
    for t in range(cfg.steps):
        q, h = wl.q(t), wl.h(t)
        kn, vn = wl.kv_new(t)
        ref = a.ctx.step(a.dev(q), a.dev(h), a.dev(kn), a.dev(vn))
        a.ctx.sync()
        to_h = (lambda x: to_torch(x, cfg.dtype).pin_memory()) if pinned_out else (lambda x: to_torch(x, cfg.dtype))
        b_.ctx.step_host(to_h(q), to_h(h) if t % 2 == 0 or t % cfg.tau == 0 else None, to_h(kn), to_h(vn), out_h)
        assert torch.equal(ref.cpu(), out_h), f"step {t}"
    for s_ in range(cfg.B):
        assert a.ctx.page_table(s_) == b_.ctx.page_table(s_)
    sa, sb = a.ctx.stats(), b_.ctx.stats()
    assert (sa["hits"], sa["misses"], sa["bytes_fetched"]) == (sb["hits"], sb["misses"], sb["bytes_fetched"])
    a.ctx.close(); b_.ctx.close()


def test_step_host_async_tickets_equal_step():
    """lsa_step_host_async (step_overlap = 1): several steps in flight, each with pinned inputs and a pinned output of its own,
    tickets waited for out of lock-step with the calls; outputs, page tables and counters must equal those of lsa_step on a
    second context fed the same inputs.  Trigger and swap steps are part of the run."""
    cfg = make_config(2, B=2, L=[16384 + 4 * 37, 8192], W=1024, k=6, hot_pages=32, steps=44, name="cfg2_host_async", q_gain=16.0, tau=8)
    wl = LsaWorkload(cfg)
    a, b_ = GpuRig(wl, step_overlap=1), GpuRig(wl, step_overlap=1)
    pinh = lambda x: to_torch(x, cfg.dtype).pin_memory()
    ins = [(pinh(wl.q(t)), pinh(wl.h(t)), pinh(wl.kv_new(t)[0]), pinh(wl.kv_new(t)[1])) for t in range(cfg.steps)]
    outs = [torch.empty((cfg.B, cfg.H, cfg.D), dtype=torch.bfloat16).pin_memory() for _ in range(cfg.steps)]
    refs, tickets = [], []
    for t in range(cfg.steps):
        q, h = wl.q(t), wl.h(t)
        kn, vn = wl.kv_new(t)
        refs.append(a.ctx.step(a.dev(q), a.dev(h), a.dev(kn), a.dev(vn)))
        tickets.append(b_.ctx.step_host_async(ins[t][0], ins[t][1], ins[t][2], ins[t][3], outs[t]))
        assert tickets[-1] > 0, "the overlapped path must hand out real tickets"
        if t >= 5 and t % 3 == 0:                       # wait for an older step while newer ones are in flight
            b_.ctx.host_wait(tickets[t - 5])
            a.ctx.sync()
            assert torch.equal(refs[t - 5].cpu(), outs[t - 5]), f"step {t - 5}"
    for t in range(cfg.steps):
        b_.ctx.host_wait(tickets[t])
    a.ctx.sync()
    for t in range(cfg.steps):
        assert torch.equal(refs[t].cpu(), outs[t]), f"step {t}"
    for s_ in range(cfg.B):
        assert a.ctx.page_table(s_) == b_.ctx.page_table(s_)
    sa, sb = a.ctx.stats(), b_.ctx.stats()
    assert (sa["hits"], sa["misses"], sa["bytes_fetched"]) == (sb["hits"], sb["misses"], sb["bytes_fetched"])
    a.ctx.close(); b_.ctx.close()


def test_recall_lag_deeper_than_one_step_flagship_shape_and_bounds():
    """recall_lag in 2..tau-1 (a longer fetch hides behind more steps; default stays the paper's t+1): lock-step on
    the tcgen05 path - the swap then rides on the attention launch lag steps after the trigger - and the init bound."""
    from paper_2606_09079_b200 import lsa
    cfg = make_config(2, B=2, L=[16384 + 4 * 37, 8192], W=1024, k=6, hot_pages=32, steps=26, name="cfg2_lag5", q_gain=16.0, tau=8,
                      recall_lag=5)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    r = run_lockstep(wl, rig, cfg.steps)
    assert r["checked"] == cfg.steps
    rig.ctx.close()
    with pytest.raises(lsa.LsaError):
        GpuRig(LsaWorkload(make_small_config("bf16", tau=4, recall_lag=4)))      # a second table would be staged before the swap


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_export_chunks_fills_the_cold_pool_bit_exactly(dtype):
    """NEXT-4, first half (P:179, P:199 VRAM -> DRAM): parts of the pinned cold pool start zeroed; lsa_export_chunks copies
    their page images from HBM (bit-exact, ragged chunk ranges), and the lock-step run that follows - whose fetches read
    the cold pool - matches the oracle, which holds the true data throughout."""
    from paper_2606_09079_b200 import lsa
    cfg = make_small_config(dtype, steps=10, q_gain=8.0)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    true = [x.clone() for x in rig.cold]
    n0, n1 = cfg.n_chunks(0), cfg.n_chunks(1)
    rig.cold[0][: n0 - 5].zero_()
    rig.cold[1].zero_()
    srcs = [true[0][:7].to(rig.device), true[0][7: n0 - 5].to(rig.device), true[1].to(rig.device)]
    torch.cuda.synchronize()
    rig.ctx.export_chunks(0, 0, srcs[0])
    rig.ctx.export_chunks(0, 7, srcs[1])
    rig.ctx.export_chunks(1, 0, srcs[2])
    rig.ctx.export_chunks(1, n1, srcs[2][:0])                       # empty range at the end: a no-op
    rig.ctx.sync()
    assert torch.equal(rig.cold[0], true[0]) and torch.equal(rig.cold[1], true[1])
    with pytest.raises(lsa.LsaError):
        rig.ctx.export_chunks(1, n1 - 1, srcs[2][:2])               # past the last chunk
    with pytest.raises(lsa.LsaError):
        rig.ctx.export_chunks(2, 0, srcs[2])                        # no such sequence
    r = run_lockstep(wl, rig, cfg.steps)
    assert r["checked"] == cfg.steps and rig.ctx.stats()["misses"] > 0
    rig.ctx.close()


def test_step_graph_replays_and_matches_oracle():
    """lsa_step_graph (NEXT-3): steps without a trigger or a table swap replay one captured CUDA graph (S6 fold,
    window append, attention, combine); trigger steps and the step that swaps the tables run as lsa_step.  Same lock-step
    checks as lsa_step: page tables / residency / fetched bytes bit-exact, attention within tolerance, every step."""
    cfg = make_config(2, B=2, L=[16384 + 4 * 37, 8192], W=1024, k=6, hot_pages=32, steps=40, name="cfg2_graph", q_gain=16.0, tau=8)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    dev = rig.device
    qd = torch.empty((cfg.B, cfg.H, cfg.D), dtype=torch.bfloat16, device=dev)
    hd = torch.empty((cfg.B, cfg.Dh), dtype=torch.bfloat16, device=dev)
    knd = torch.empty((cfg.B, cfg.D), dtype=torch.bfloat16, device=dev)
    vnd = torch.empty_like(knd)
    outd = torch.empty_like(qd)

    def step_fn(q, h, kn, vn):
        rig.ctx.sync()                                   # the previous step has finished reading the fixed buffers
        qd.copy_(rig.dev(q)); hd.copy_(rig.dev(h)); knd.copy_(rig.dev(kn)); vnd.copy_(rig.dev(vn))
        torch.cuda.synchronize()                         # the library's streams are not torch's current stream
        return rig.ctx.step_graph(qd, hd, knd, vnd, outd)

    r = run_lockstep(wl, rig, cfg.steps, step_fn=step_fn)
    assert r["checked"] == cfg.steps
    gs = rig.ctx.graph_stats()
    # 40 steps, tau = 8: 5 trigger steps + 5 swap steps run plain; the other 30 share ONE graph (window full: fixed geometry)
    assert gs["captures"] == 1 and gs["replays"] == 29, gs
    rig.ctx.close()


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("lag", [0, 1, 3])
def test_lockstep_small(dtype, lag):
    cfg = make_small_config(dtype, recall_lag=lag, steps=14, q_gain=8.0)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    r = run_lockstep(wl, rig, cfg.steps)
    assert r["checked"] == cfg.steps


@pytest.mark.parametrize("max_ctas", [1, 3, 0])
def test_lockstep_small_split_counts(max_ctas):
    """Split-K geometry must not change results: 1 split, 3 splits, one full wave."""
    cfg = make_small_config("f32", steps=6, q_gain=8.0)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl, max_ctas=max_ctas)
    run_lockstep(wl, rig, cfg.steps)


def test_k_equals_all_chunks_is_dense_attention():
    cfg = make_small_config("f32", B=2, L=[2048, 1216], k=32, hot_pages=128, recall_lag=0, tau=4, q_gain=8.0)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    q = wl.q(0)
    out = rig.host(rig.ctx.step(rig.dev(q), rig.dev(wl.h(0))))
    for b in range(cfg.B):
        ncsa = cfg.n_csa(b)
        cold = as_f64(wl.cold_csa[b], "f32")
        Kd = np.concatenate([as_f64(wl.hca_k[b], "f32"), cold[:, 0].reshape(-1, cfg.D)[:ncsa], as_f64(wl.win_k[b], "f32")])
        Vd = np.concatenate([as_f64(wl.hca_v[b], "f32"), cold[:, 1].reshape(-1, cfg.D)[:ncsa], as_f64(wl.win_v[b], "f32")])
        ref = torch.nn.functional.scaled_dot_product_attention(
            torch.from_numpy(as_f64(q[b], "f32"))[None], torch.from_numpy(Kd)[None], torch.from_numpy(Vd)[None],
            scale=1 / math.sqrt(cfg.D))[0].numpy()
        np.testing.assert_allclose(out[b], ref, atol=1e-4, rtol=1e-4)


# ------------------------------------------------------------------------------- BASELINE configs
def test_cfg1_every_step():
    wl = LsaWorkload(make_config(1))
    rig = GpuRig(wl)
    r = run_lockstep(wl, rig, wl.cfg.steps)
    assert r["checked"] == 128
    st = rig.ctx.stats()
    assert st["triggers"] == 2 and st["misses"] == 4 and st["hits"] == 4


def _sample_steps(cfg, steps):
    s = set()
    for t in range(steps):
        if t % cfg.tau == 0 or t % cfg.tau == 1 or t % 64 == 37:
            s.add(t)
    return s


def test_cfg2_sampled():
    wl = LsaWorkload(make_config(2))
    rig = GpuRig(wl)
    steps = 64 * 9 + 2                      # crosses two needle-drift epochs (every 4 triggers)
    r = run_lockstep(wl, rig, steps, check_attention_at=_sample_steps(wl.cfg, steps))
    assert r["checked"] >= 27


def test_cfg3_sampled_bench_launch_config():
    wl = LsaWorkload(make_config(3))
    rig = GpuRig(wl)
    steps = 64 * 5 + 2
    r = run_lockstep(wl, rig, steps, check_attention_at=_sample_steps(wl.cfg, steps))
    assert r["checked"] >= 15
    assert rig.ctx.stats()["misses"] >= 64


def test_cfg5_churn_sampled():
    cfg = make_config(5)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    steps = 16 * 6 + 2                      # the seeded draws mark sequence 2's triggers 5 and 6 (steps 80 and 96) as tie triggers
    r = run_lockstep(wl, rig, steps, check_attention_at={0, 1, 16, 17, 33, 64, 65, 81, 97})
    st = rig.ctx.stats()
    assert st["evictions"] > 0 and st["misses"] > 3 * 8 * 128 * 0.6
    # BASELINE.json configs[4]: 10 % of the triggers carry a planted exact tie and a one-ulp near-tie across the k-th rank
    assert r["tie_triggers"] >= 2


def test_cfg4_ragged_batch_sampled():
    cfg = make_config(4)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    steps = 70
    r = run_lockstep(wl, rig, steps, check_attention_at={0, 1, 3, 63, 64, 65, 69})
    assert rig.ctx.stats()["triggers"] == 32 + 3      # every sequence once, sequences 0..2 twice


# ------------------------------------------------------------------------------- S7-S8, small batches (lsa_attn_tc_small.cuh)
@pytest.mark.parametrize("overlap", [0, 1])
@pytest.mark.parametrize("max_ctas", [0, 3, 7])
def test_small_batch_half_tile_split_edge_cases(max_ctas, overlap):
    """B <= 4 on the tensor-core path: pieces are cut at 64-row half tiles.  Row counts around the 64 / 128
    boundaries in the HCA and window segments, cut by 3, 7 and one CTA per SM, so that lone halves, merged
    halves and ragged tails all occur at piece starts and ends; every sequence against the oracle's attention."""
    lsa = _lsa()
    dev = torch.device("cuda:0")
    H, D, W = 64, 512, 400
    g = torch.Generator().manual_seed(31)
    rnd = lambda *s: torch.randn(*s, generator=g).to(torch.bfloat16).to(dev)
    for n_rows, w_len in [([63, 64, 65, 127], [1, 64, 65, 0]), ([128, 129, 191, 192], [127, 128, 129, 193]),
                          ([1000], [333]), ([0, 257], [64, 0]), ([5, 0, 70], [0, 0, 300])]:
        B = len(n_rows)
        hk, hv = [rnd(n, D) for n in n_rows], [rnd(n, D) for n in n_rows]
        wk, wv = [rnd(W, D) for _ in range(B)], [rnd(W, D) for _ in range(B)]
        q = rnd(B, H, D)
        ctx = _direct_ctx("bf16", H, D, 128, hk, hv, wk, wv, w_len, W, sm_scale=0.08, max_ctas=max_ctas,
                          attn_impl=lsa.LSA_ATTN_TCGEN05, step_overlap=overlap)
        for rep in range(3):
            out, lse = ctx.decode_attention(q, want_lse=True)
        ctx.sync()
        out64, lse = out.double().cpu().numpy(), lse.cpu().numpy()
        for b in range(B):
            K = np.concatenate([hk[b].double().cpu().numpy(), wk[b][: w_len[b]].double().cpu().numpy()])
            V = np.concatenate([hv[b].double().cpu().numpy(), wv[b][: w_len[b]].double().cpu().numpy()])
            if len(K) == 0:
                assert torch.all(out[b] == 0) and np.all(lse[b] == -np.inf)
                continue
            ref, ref_lse, _ = attention(q[b].double().cpu().numpy(), K, V, 0.08)
            np.testing.assert_allclose(out64[b], ref, err_msg=f"rows {n_rows} w_len {w_len} seq {b}", **attn_tolerance("bf16"))
            np.testing.assert_allclose(lse[b], ref_lse, atol=2e-2, rtol=1e-3)
        ctx.close()


@pytest.mark.parametrize("overlap", [0, 1])
def test_small_batch_steps_back_to_back_without_sync(overlap):
    """The small-batch launches do not wait for the previous step's merge (partials in rotating workspace buffers, the ring row
    ordered by SeqDev::app_epoch): 48 steps of two contexts interleaved on one stream, each with its own q and its
    own output buffer, no host synchronisation in between; every output is then compared with the oracle, which
    sees the window grow by one row per step."""
    lsa = _lsa()
    dev = torch.device("cuda:0")
    H, D, W, steps = 64, 512, 640, 48
    g = torch.Generator().manual_seed(32)
    rnd = lambda *s: torch.randn(*s, generator=g).to(torch.bfloat16).to(dev)
    st = torch.cuda.Stream(dev)
    rigs = []
    for n_rows, w_len in [([900, 300], [600, 61]), ([2000], [127])]:
        B = len(n_rows)
        hk, hv = [rnd(n, D) for n in n_rows], [rnd(n, D) for n in n_rows]
        wk, wv = [rnd(W, D) for _ in range(B)], [rnd(W, D) for _ in range(B)]
        w0k, w0v = [x.clone() for x in wk], [x.clone() for x in wv]
        lsa_mod = lsa
        seqs = [dict(cold_csa=None, n_csa=0, chunk_emb=None, hca_k=hk[b], hca_v=hv[b], win_k=wk[b], win_v=wv[b], w_len=w_len[b],
                     w_head=w_len[b] % W, step0=1) for b in range(B)]
        ctx = lsa_mod.LsaContext(dtype=1, H=H, D=D, C_=128, W=W, Dh=64, E=64, k=1, tau=1 << 20, sm_scale=0.06,
                                 hot_pool=torch.zeros((2 * B, 2, 128, D), dtype=torch.bfloat16, device=dev),
                                 W_q=torch.zeros((64, 64), dtype=torch.bfloat16, device=dev), seqs=seqs, stream_compute=st,
                                 attn_impl=lsa.LSA_ATTN_TCGEN05, step_overlap=overlap)
        rigs.append(dict(ctx=ctx, B=B, hk=hk, hv=hv, w0k=w0k, w0v=w0v, w_len=w_len,
                         q=[rnd(B, H, D) for _ in range(steps)], kn=[rnd(B, D) for _ in range(steps)], vn=[rnd(B, D) for _ in range(steps)],
                         out=[torch.empty((B, H, D), dtype=torch.bfloat16, device=dev) for _ in range(steps)]))
    torch.cuda.synchronize()
    for t in range(steps):
        for r in rigs:
            r["ctx"].step(r["q"][t], None, r["kn"][t], r["vn"][t], r["out"][t])
    st.synchronize()
    tol = attn_tolerance("bf16")
    for r in rigs:
        wk = [x.double().cpu().numpy().copy() for x in r["w0k"]]
        wv = [x.double().cpu().numpy().copy() for x in r["w0v"]]
        w_len, head = list(r["w_len"]), [w % W for w in r["w_len"]]
        for t in range(steps):
            for b in range(r["B"]):
                wk[b][head[b]] = r["kn"][t][b].double().cpu().numpy()
                wv[b][head[b]] = r["vn"][t][b].double().cpu().numpy()
                head[b] = (head[b] + 1) % W
                w_len[b] = min(W, w_len[b] + 1)
                K = np.concatenate([r["hk"][b].double().cpu().numpy(), wk[b][: w_len[b]]])
                V = np.concatenate([r["hv"][b].double().cpu().numpy(), wv[b][: w_len[b]]])
                ref, _, _ = attention(r["q"][t][b].double().cpu().numpy(), K, V, 0.06)
                np.testing.assert_allclose(r["out"][t][b].double().cpu().numpy(), ref, err_msg=f"step {t} seq {b}", **tol)
        r["ctx"].close()


@pytest.mark.parametrize("max_ctas,n_rows,w_len", [(0, [11200], [900]), (40, [3333], [1100]), (100, [11000], [1000]),
                                                   (100, [7000, 5000], [1000, 160]), (0, [3000, 2000, 1500, 800], [500, 64, 0, 129])])
def test_small_batch_last_arrivals_merge(max_ctas, n_rows, w_len):
    """S8 of the small-batch kernel (step_overlap = 1): only the launch's last arrivals merge, the other CTAs leave.
    Shapes and CTA caps that give (a) 48 CTAs with 32 mergers of one round each, (b) 36 CTAs and a ragged last piece,
    (c) 94 CTAs: more than 64 partial slots (3 boxes of 32 slots, 4 units per round), 32 mergers of two rounds each beside
    62 leavers, (d) two sequences: 16 units per merger, (e) four sequences: every CTA merges, four rounds each.  Seven
    launches back to back walk twice through the three workspace buffers; every output against the oracle's attention."""
    lsa = _lsa()
    dev = torch.device("cuda:0")
    H, D, W = 64, 512, 1200
    g = torch.Generator().manual_seed(41)
    rnd = lambda *s: torch.randn(*s, generator=g).to(torch.bfloat16).to(dev)
    B = len(n_rows)
    hk, hv = [rnd(n, D) for n in n_rows], [rnd(n, D) for n in n_rows]
    wk, wv = [rnd(W, D) for _ in range(B)], [rnd(W, D) for _ in range(B)]
    qs = [rnd(B, H, D) for _ in range(7)]
    ctx = _direct_ctx("bf16", H, D, 128, hk, hv, wk, wv, w_len, W, sm_scale=0.05, max_ctas=max_ctas,
                      attn_impl=lsa.LSA_ATTN_TCGEN05, step_overlap=1)
    res = [ctx.decode_attention(q, want_lse=True) for q in qs]      # no synchronisation in between
    ctx.sync()
    for q, (out, lse) in zip(qs, res):
        for b in range(B):
            K = np.concatenate([hk[b].double().cpu().numpy(), wk[b][: w_len[b]].double().cpu().numpy()])
            V = np.concatenate([hv[b].double().cpu().numpy(), wv[b][: w_len[b]].double().cpu().numpy()])
            ref, ref_lse, _ = attention(q[b].double().cpu().numpy(), K, V, 0.05)
            np.testing.assert_allclose(out[b].double().cpu().numpy(), ref, err_msg=f"seq {b}", **attn_tolerance("bf16"))
            np.testing.assert_allclose(lse[b].cpu().numpy(), ref_lse, atol=2e-2, rtol=1e-3)
    ctx.close()


@pytest.mark.parametrize("overlap", [0, 1])
def test_small_batch_merge_never_multiplies_a_foreign_slot(overlap):
    """Partial slot = CTA + sequence, so the slots a sequence's merge walks include other sequences' partials (weight 0).
    They are selected away, not multiplied: a NaN fed into sequence 0 leaves sequence 1's output exact
    (step_overlap 1: the in-launch merge; 0: the large-grid kernel + combine kernel)."""
    lsa = _lsa()
    dev = torch.device("cuda:0")
    H, D, W = 64, 512, 700
    g = torch.Generator().manual_seed(47)
    rnd = lambda *s: torch.randn(*s, generator=g).to(torch.bfloat16).to(dev)
    n_rows, w_len = [5000, 4000], [600, 333]
    hk, hv = [rnd(n, D) for n in n_rows], [rnd(n, D) for n in n_rows]
    wk, wv = [rnd(W, D) for _ in range(2)], [rnd(W, D) for _ in range(2)]
    hv[0][1234, 77] = float("nan")
    hk[0][4000, 5] = float("nan")
    q = rnd(2, H, D)
    ctx = _direct_ctx("bf16", H, D, 128, hk, hv, wk, wv, w_len, W, sm_scale=0.05, attn_impl=lsa.LSA_ATTN_TCGEN05, step_overlap=overlap)
    outs = [ctx.decode_attention(q) for _ in range(5)]
    ctx.sync()
    K = np.concatenate([hk[1].double().cpu().numpy(), wk[1][: w_len[1]].double().cpu().numpy()])
    V = np.concatenate([hv[1].double().cpu().numpy(), wv[1][: w_len[1]].double().cpu().numpy()])
    ref, _, _ = attention(q[1].double().cpu().numpy(), K, V, 0.05)
    for out in outs:                                  # (what sequence 0 itself gets for NaN inputs is not specified)
        assert torch.isfinite(out[1]).all()
        np.testing.assert_allclose(out[1].double().cpu().numpy(), ref, **attn_tolerance("bf16"))
    ctx.close()


def test_small_batch_timeline():
    """lsa_timeline_*: every CTA of a stamped launch has ordered stamps, the launch's last 32 arrivals (all of them if it has
    fewer CTAs) carry merger stamps, and stamping does not change the result."""
    lsa = _lsa()
    dev = torch.device("cuda:0")
    H, D, W = 64, 512, 1200
    g = torch.Generator().manual_seed(43)
    rnd = lambda *s: torch.randn(*s, generator=g).to(torch.bfloat16).to(dev)
    hk, hv, wk, wv = [rnd(11200, D)], [rnd(11200, D)], [rnd(W, D)], [rnd(W, D)]
    q = rnd(1, H, D)
    ctx = _direct_ctx("bf16", H, D, 128, hk, hv, wk, wv, [900], W, sm_scale=0.05, attn_impl=lsa.LSA_ATTN_TCGEN05, step_overlap=1)
    ref = ctx.decode_attention(q)
    tl0, n0 = ctx.timeline_read()                                 # (waits for both streams)
    assert n0 == 0 and not tl0.any()
    ctx.timeline_enable(True)
    outs = [ctx.decode_attention(q) for _ in range(5)]            # an output buffer each
    ctx.timeline_enable(False)
    ctx.decode_attention(q)                                       # not stamped
    tl, n = ctx.timeline_read()
    assert n == 5
    for o in outs:
        assert torch.equal(o, ref)
    E = {name: i for i, name in enumerate(ctx.TL_EVENTS)}
    for l in range(5):
        rec = tl[l].astype(np.int64)
        n_cta = int(rec[0, E["n_ctas"]])
        assert n_cta == 48 and (rec[:n_cta, E["seq"]] == l).all() and not rec[n_cta:].any()
        r = rec[:n_cta]
        for a_, b_ in [("entry", "setup"), ("entry", "first_s"), ("first_s", "last_pv"), ("last_pv", "epilogue"), ("epilogue", "arrived"), ("arrived", "exit")]:
            assert (r[:, E[a_]] <= r[:, E[b_]]).all(), (a_, b_)
        mrg = r[:, E["merged"]] > 0
        assert mrg.sum() == 32
        assert (r[mrg, E["arrived"]] <= r[mrg, E["all_arrived"]]).all() and (r[mrg, E["all_arrived"]] <= r[mrg, E["merged"]]).all()
        assert (r[mrg, E["merged"]] <= r[mrg, E["exit"]]).all() and (r[~mrg, E["all_arrived"]] == 0).all()
        # the mergers are the LAST arrivals (a stamp is taken after the arrival, so two near-simultaneous ones may swap)
        assert r[mrg, E["arrived"]].min() + 2000 >= r[~mrg, E["arrived"]].max()
        assert (r[:, E["smid"]] < 256).all()
    assert not tl[5:].any()
    ctx.close()


def test_small_batch_step_overlap_lockstep():
    """lsa_config.step_overlap = 1 (inputs independent of the previous step's output): the whole path in lock-step with
    the oracle over several trigger periods - triggers, swaps (serialised launches) and the overlapped steps between them."""
    cfg = make_config(2, B=2, L=[16384 + 4 * 37, 8192], W=1024, k=6, hot_pages=32, steps=40, name="cfg2_overlap", q_gain=16.0, tau=8)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl, step_overlap=1)
    r = run_lockstep(wl, rig, cfg.steps)
    assert r["checked"] == cfg.steps
    rig.ctx.close()


# ---- NEXT-4 second half: the compressed history grows while decoding (DESIGN R29-R33) ------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("lag", [0, 1, 2])
def test_growth_lockstep_small_f32(lag):
    """SIMT path, every step checked: a CSA entry every step, an HCA entry every 16, chunks of 16 entries, so in 200 steps 12
    chunks per sequence complete, are exported, become candidates and some are recalled again from their cold copy.  The
    window (24 rows) wraps 8 times: the decoded tokens really move from the window into CSA / HCA entries."""
    from lsa_harness import GrowthRig, run_growth_lockstep
    from paper_2606_09079_b200.workloads import GrowthInputs
    cfg = make_small_config("f32", B=2, L=[4096 + 24, 2432], C=16, W=24, k=5, tau=4, steps=0, hot_pages=20, needle_period=10 ** 9,
                            recall_lag=lag)
    wl = LsaWorkload(cfg)
    gi = GrowthInputs(wl, steps=200, csa_every=1, hca_every=16, hot_frac=1.0)
    rig = GrowthRig(wl, gi)
    res = run_growth_lockstep(wl, gi, rig, 200)
    assert res["checked"] == 200 and res["exported"] >= 24 and res["recalled_grown"] > 0
    assert res["csa_appended"] == 2 * 199 and res["hca_appended"] == 2 * 12


@pytest.mark.gpu
@pytest.mark.parametrize("overlap", [0, 1])
def test_growth_lockstep_tcgen05(overlap):
    """Tensor-core path at the BASELINE shape (bf16, H 64, D 512, C 128) with the paper's cadences (one CSA entry per 4 tokens,
    one HCA entry per 128), 1100 steps > W = 512: two chunks complete per sequence; B = 2 with a ragged start (one sequence
    begins inside a chunk).  step_overlap 1 takes the small-batch kernel, 0 the large-grid kernel + combine."""
    from lsa_harness import GrowthRig, run_growth_lockstep
    from paper_2606_09079_b200.workloads import GrowthInputs
    cfg = make_small_config("bf16", B=2, L=[32768 + 4 * 50, 16384], H=64, D=512, C=128, W=512, Dh=256, E=128, k=6, tau=64,
                            steps=0, hot_pages=24, needle_period=10 ** 9, n_needles=3)
    wl = LsaWorkload(cfg)
    gi = GrowthInputs(wl, steps=1100, csa_every=4, hca_every=128, hot_frac=1.0)
    rig = GrowthRig(wl, gi, step_overlap=overlap)
    check = set(range(0, 1100, 37)) | set(range(300, 330)) | set(range(508, 520)) | {1099}
    res = run_growth_lockstep(wl, gi, rig, 1100, check_attention_at=check, check_tables_every=16)
    assert res["exported"] == 2 + 2 and res["csa_appended"] == 2 * 274 and res["hca_appended"] == 2 * 8
    from paper_2606_09079_b200 import lsa
    assert rig.ctx.stats()["attn_impl"] == lsa.LSA_ATTN_TCGEN05


@pytest.mark.gpu
def test_growth_argument_errors():
    from paper_2606_09079_b200 import lsa
    from lsa_harness import GrowthRig, GpuRig
    from paper_2606_09079_b200.workloads import GrowthInputs
    cfg = make_small_config("f32", B=2, L=[4096, 2432], C=16, W=24, k=5, tau=4, steps=0, hot_pages=20, needle_period=10 ** 9)
    wl = LsaWorkload(cfg)
    gi = GrowthInputs(wl, steps=8, csa_every=1)
    rig = GrowthRig(wl, gi)
    z = torch.zeros((2, cfg.D), device="cuda")
    with pytest.raises(lsa.LsaError):                       # a pair must be complete
        rig.ctx.append_compressed([0, 1], csa_k=z)
    with pytest.raises(lsa.LsaError):                       # ids ascending
        rig.ctx.append_compressed([1, 0], csa_k=z, csa_v=z)
    for _ in range(15):
        rig.ctx.append_compressed([0, 1], csa_k=z, csa_v=z)
    with pytest.raises(lsa.LsaError):                       # the 16th entry completes a chunk: emb_rows required
        rig.ctx.append_compressed([0, 1], csa_k=z, csa_v=z)
    rig.ctx.append_compressed([0, 1], csa_k=z, csa_v=z, emb_rows=torch.zeros((2, cfg.E), device="cuda"))
    with pytest.raises(lsa.LsaError):                       # capacity: cap_csa = n_csa + 8 + 1 rounded up to a chunk
        for _ in range(40):
            rig.ctx.append_compressed([0, 1], csa_k=z, csa_v=z, emb_rows=torch.zeros((2, cfg.E), device="cuda"))
    static = GpuRig(LsaWorkload(make_small_config("f32")))
    with pytest.raises(lsa.LsaError):                       # a context without capacity cannot grow
        static.ctx.append_compressed([0], csa_k=z[:1], csa_v=z[:1])
