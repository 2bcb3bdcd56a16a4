"""Glue shared by the tests: build the oracle (and, on a GPU, the CUDA context) from one
seeded workload.  Lives in tests/ because only tests may touch oracle/."""
from __future__ import annotations

import numpy as np

from oracle import LsaOracle
from paper_2606_09079_b200.workloads import LsaWorkload


def make_oracle(wl: LsaWorkload, trigger_idx: int = 0, **over) -> LsaOracle:
    c = wl.cfg
    kw = dict(
        dtype=c.dtype, H=c.H, D=c.D, C=c.C, W=c.W, k=c.k, tau=c.tau, recall_lag=c.recall_lag,
        hot_pages=c.hot_pages, W_q=wl.W_q, cold_csa=wl.cold_csa,
        n_csa=[c.n_csa(b) for b in range(c.B)],
        chunk_emb=[wl.chunk_emb(b, trigger_idx) for b in range(c.B)],
        hca_k=wl.hca_k, hca_v=wl.hca_v, win_k=wl.win_k, win_v=wl.win_v,
        w_len=[min(c.W, c.L[b]) for b in range(c.B)], w_head=[min(c.W, c.L[b]) % c.W for b in range(c.B)],
        step0=[c.step0(b) for b in range(c.B)])
    kw.update(over)
    return LsaOracle(**kw)


def growth_arrays(wl: LsaWorkload, gi):
    """Capacity-sized copies of the workload's arrays for a run whose compressed history grows (NEXT-4): the cold pool,
    the embedding table and the HCA arrays with room for what `gi` (workloads.GrowthInputs) will hand over."""
    c = wl.cfg
    cold, emb, hk, hv = [], [], [], []
    for b in range(c.B):
        cap_ch = gi.cap_csa(b) // c.C
        x = np.zeros((cap_ch,) + wl.cold_csa[b].shape[1:], dtype=wl.cold_csa[b].dtype)
        x[: c.n_chunks(b)] = wl.cold_csa[b]
        cold.append(x)
        e0 = wl.chunk_emb(b, 0)
        e = np.zeros((cap_ch, c.E), dtype=e0.dtype)
        e[: c.n_chunks(b)] = e0
        emb.append(e)
        for src, dst in ((wl.hca_k[b], hk), (wl.hca_v[b], hv)):
            y = np.zeros((gi.cap_hca(b), c.D), dtype=src.dtype)
            y[: c.n_hca(b)] = src
            dst.append(y)
    return cold, emb, hk, hv


def make_growing_oracle(wl: LsaWorkload, gi, **over):
    from oracle.growth_oracle import GrowingLsaOracle
    c = wl.cfg
    cold, emb, hk, hv = growth_arrays(wl, gi)
    kw = dict(
        dtype=c.dtype, H=c.H, D=c.D, C=c.C, W=c.W, k=c.k, tau=c.tau, recall_lag=c.recall_lag,
        hot_pages=c.hot_pages, W_q=wl.W_q, cold_csa=cold, n_csa=[c.n_csa(b) for b in range(c.B)],
        n_hca=[c.n_hca(b) for b in range(c.B)], chunk_emb=emb, hca_k=hk, hca_v=hv, win_k=wl.win_k, win_v=wl.win_v,
        w_len=[min(c.W, c.L[b]) for b in range(c.B)], w_head=[min(c.W, c.L[b]) % c.W for b in range(c.B)],
        step0=[c.step0(b) for b in range(c.B)])
    kw.update(over)
    return GrowingLsaOracle(**kw)


def oracle_appends(orc, gi, t: int):
    """Hand the entries due before decode step t to the oracle (R29).  Returns [(b, chunk)] completed by them."""
    c = orc
    done = []
    hca = gi.hca_entry(t) if gi.hca_due(t) else None
    csa = gi.csa_entry(t) if gi.csa_due(t) else None
    if hca is None and csa is None:
        return done
    for b in range(orc.B):
        emb_row = None
        if csa is not None and orc.n_csa[b] % orc.C == orc.C - 1:
            emb_row = gi.emb_row(b, orc.n_csa[b] // orc.C)
        if orc.append_compressed(b, None if csa is None else csa[0][b], None if csa is None else csa[1][b],
                                 None if hca is None else hca[0][b], None if hca is None else hca[1][b], emb_row):
            done.append((b, orc.n_chunks[b] - 1))
    return done


def apply_emb_updates(wl: LsaWorkload, oracle: LsaOracle, global_step: int, gpu_embs=None):
    """Needle drift (cfg 2-4): rewrite embedding rows before the trigger at `global_step`."""
    import torch
    from paper_2606_09079_b200.workloads import to_torch
    c = wl.cfg
    for b in range(c.B):
        if not wl.fires(b, global_step):
            continue
        upd = wl.emb_row_updates(b, wl.trigger_index(b, global_step))
        if upd is None:
            continue
        ids, rows = upd
        oracle.chunk_emb[b] = oracle.chunk_emb[b].copy()
        oracle.chunk_emb[b][ids] = rows
        if gpu_embs is not None:
            gpu_embs[b][torch.from_numpy(ids).to(gpu_embs[b].device)] = to_torch(rows, c.dtype).to(gpu_embs[b].device)


# ------------------------------------------------------------------------------------------
# GPU side (only used by -m gpu tests and smoke)
# ------------------------------------------------------------------------------------------
class GpuRig:
    """Device / pinned tensors of one workload plus the LsaContext built on them."""

    def __init__(self, wl: LsaWorkload, trigger_idx: int = 0, device="cuda:0", **ctx_over):
        import torch
        from paper_2606_09079_b200 import lsa
        from paper_2606_09079_b200.workloads import to_torch
        c = wl.cfg
        self.wl, self.cfg, self.device = wl, c, torch.device(device)
        dt = c.dtype
        tdt = torch.float32 if dt == "f32" else torch.bfloat16
        dev = self.device
        self.hot_pool = torch.zeros((c.hot_pages, 2, c.C, c.D), dtype=tdt, device=dev)
        self.W_q = to_torch(wl.W_q, dt).to(dev)
        self.cold = [to_torch(x, dt).pin_memory() for x in wl.cold_csa]
        self.emb = [to_torch(wl.chunk_emb(b, trigger_idx), dt).to(dev) for b in range(c.B)]
        self.hca_k = [to_torch(x, dt).to(dev) for x in wl.hca_k]
        self.hca_v = [to_torch(x, dt).to(dev) for x in wl.hca_v]
        self.win_k = [to_torch(x, dt).to(dev) for x in wl.win_k]
        self.win_v = [to_torch(x, dt).to(dev) for x in wl.win_v]
        seqs = []
        for b in range(c.B):
            seqs.append(dict(cold_csa=self.cold[b], n_csa=c.n_csa(b), chunk_emb=self.emb[b],
                             hca_k=self.hca_k[b], hca_v=self.hca_v[b], win_k=self.win_k[b], win_v=self.win_v[b],
                             w_len=min(c.W, c.L[b]), w_head=min(c.W, c.L[b]) % c.W, step0=c.step0(b)))
        kw = dict(dtype=lsa.LSA_F32 if dt == "f32" else lsa.LSA_BF16, H=c.H, D=c.D, C_=c.C, W=c.W, Dh=c.Dh, E=c.E,
                  k=c.k, tau=c.tau, hot_pool=self.hot_pool, W_q=self.W_q, seqs=seqs, recall_lag=c.recall_lag)
        kw.update(ctx_over)
        self.ctx = lsa.LsaContext(**kw)
        self.tdt = tdt

    def dev(self, arr):
        from paper_2606_09079_b200.workloads import to_torch
        return to_torch(arr, self.cfg.dtype).to(self.device)

    def host(self, t):
        from paper_2606_09079_b200.workloads import as_f64, from_torch
        self.ctx.sync()          # the library's streams are not torch's current stream
        return as_f64(from_torch(t, self.cfg.dtype), self.cfg.dtype)


def attn_tolerance(dtype: str):
    """BASELINE.json north_star: abs 2e-2 / rel 1e-2 for bf16 inputs, 1e-4 for the fp32 config."""
    return dict(atol=2e-2, rtol=1e-2) if dtype == "bf16" else dict(atol=1e-4, rtol=1e-4)


def apply_tie_triggers(wl: LsaWorkload, oracle: LsaOracle, rig, global_step: int, h, state: dict) -> int:
    """BASELINE.json cfg 5: "10% of triggers carry planted exact-tie and near-tie scores".  At a trigger the workload marks
    (LsaWorkload.has_tie_trigger) both sides get the table in force with an exact tie planted across the k-th rank of the
    ORACLE's ranking (rank k+1's row becomes a bit copy of rank k's: the lower chunk id must win) and a one-ulp near-tie
    behind it; the next trigger of that sequence restores the plain table.  Returns the number of tie triggers applied."""
    from oracle import chunk_scores, query_tower
    from paper_2606_09079_b200.workloads import plant_boundary_ties, to_torch
    c = wl.cfg
    n = 0
    for b in range(c.B):
        if not wl.fires(b, global_step):
            continue
        trig = wl.trigger_index(b, global_step)
        if wl.has_tie_trigger(b, trig):
            base = state.get(("plain", b), oracle.chunk_emb[b])
            state[("plain", b)] = base
            sc = chunk_scores(query_tower(oracle.W_q, h[b]), base)
            order = np.array(sorted(range(len(sc)), key=lambda ch: (-sc[ch], ch)))
            tied = plant_boundary_ties(base, order, c.k_eff(b), c.dtype)
            oracle.chunk_emb[b] = tied
            if rig is not None:
                t = to_torch(tied, c.dtype).to(rig.device)
                state[("dev", b)] = t                       # keep the tensor alive while the library reads it
                rig.ctx.set_chunk_emb(b, t)
            n += 1
        elif ("plain", b) in state:
            oracle.chunk_emb[b] = state.pop(("plain", b))
            if rig is not None:
                rig.ctx.set_chunk_emb(b, rig.emb[b])
    return n


def run_lockstep(wl: LsaWorkload, rig: "GpuRig", steps: int, check_attention_at=None, with_kv_new: bool = True,
                 l1=None, l1_band: float = 3e-2, step_fn=None, oracle=None):
    """Drive lsa_step and the oracle in lock-step: validate the GPU's
    selection against the oracle's scores, feed it to the oracle's residency model, then compare page
    tables / residency / fetched bytes bit-exactly and attention outputs within tolerance."""
    import torch
    from oracle import validate_selection
    c = wl.cfg
    orc = make_oracle(wl) if oracle is None else oracle
    tol = attn_tolerance(c.dtype)
    n_checked, max_err, n_ties, tie_state = 0, 0.0, 0, {}
    for t in range(steps):
        apply_emb_updates(wl, orc, t, rig.emb)
        q, h = wl.q(t), wl.h(t)
        if c.tie_frac > 0:
            n_ties += apply_tie_triggers(wl, orc, rig, t, h, tie_state)
        kn, vn = wl.kv_new(t) if with_kv_new else (None, None)
        firing = [b for b in range(c.B) if orc.step[b] % c.tau == 0]
        bytes_before = rig.ctx.stats()["bytes_fetched"] if not firing else None
        if step_fn is not None:               # another entry point with lsa_step's semantics (e.g. lsa_step_graph)
            out_gpu = step_fn(q, h, kn, vn)
        else:
            out_gpu = rig.ctx.step(rig.dev(q), rig.dev(h), None if kn is None else rig.dev(kn),
                                   None if vn is None else rig.dev(vn))
        forced = {}
        for b in firing:                      # GPU selection = chunk ids of the table it just staged
            which = 0 if c.recall_lag == 0 else 1
            chunks, pages = rig.ctx.page_table(b, which)
            import numpy as _np
            if l1 is not None:            # paper-exact Level-1 indexer drives the step (lsa_set_indexer)
                from oracle.l1_oracle import l1_index_select, validate_l1_selection
                _, _, cs, _ = l1_index_select(h[b], l1.layers, l1.index_k[b], l1.n_h, c.C, c.k)
                padded = _np.full(c.k, -1, dtype=_np.int64); padded[: len(chunks)] = chunks
                msg = validate_l1_selection(padded, cs, c.k, 0.5, l1_band)
            else:
                sc = orc.scores(b, h[b])
                order = sorted(chunks, key=lambda ch: (-sc[ch], ch))
                padded = _np.full(c.k, -1, dtype=_np.int64); padded[: len(order)] = order
                msg = validate_selection(padded, sc, c.k)
            assert msg is None, f"step {t} seq {b}: {msg}"
            forced[b] = chunks
        orc.step_begin(h, forced_selection=forced if firing else None)
        for b in firing:
            which = 0 if c.recall_lag == 0 else 1
            chunks, pages = rig.ctx.page_table(b, which)
            ref = orc.pool.cur[b] if c.recall_lag == 0 else orc.pool.nxt[b]
            assert list(zip(chunks, pages)) == ref, f"step {t} seq {b}: page table mismatch"
            assert rig.ctx.residency(b, c.n_chunks(b)) == orc.pool.page_of[b], f"step {t} seq {b}: residency mismatch"
        if firing:
            st = rig.ctx.stats()
            assert (st["hits"], st["misses"], st["evictions"], st["bytes_fetched"], st["pool_error"]) == \
                   (orc.pool.hits, orc.pool.misses, orc.pool.evictions, orc.pool.bytes_fetched, 0), f"step {t}: counters"
            hot = rig.hot_pool.cpu()
            from paper_2606_09079_b200.workloads import from_torch
            hot_np = from_torch(hot, c.dtype)
            owned = [p for p, o in enumerate(orc.pool.owner) if o is not None]
            assert _np.array_equal(hot_np[owned], orc.pool.hot[owned]), f"step {t}: fetched bytes differ"
        else:
            assert rig.ctx.stats()["bytes_fetched"] == bytes_before      # P:185 zero transfers inside a window
        attend = check_attention_at is None or t in check_attention_at
        res = orc.step_end(q, kn, vn, attend=attend)
        if attend:
            got = rig.host(out_gpu)
            import numpy as np
            np.testing.assert_allclose(got, res[0], err_msg=f"attention mismatch at step {t}", **tol)
            max_err = max(max_err, float(np.max(np.abs(got - res[0]))))
            n_checked += 1
    rig.ctx.sync()
    return dict(checked=n_checked, max_abs_err=max_err, oracle=orc, tie_triggers=n_ties)


# ------------------------------------------------------------------------------------------
# NEXT-4 second half: lock-step run with a growing compressed history
# ------------------------------------------------------------------------------------------
class GrowthRig(GpuRig):
    """GpuRig whose per-sequence arrays have the capacity GrowthInputs asks for (lsa_seq_desc.cap_csa / cap_hca)."""

    def __init__(self, wl: LsaWorkload, gi, device="cuda:0", **ctx_over):
        import torch
        from paper_2606_09079_b200 import lsa
        from paper_2606_09079_b200.workloads import to_torch
        c = wl.cfg
        self.wl, self.cfg, self.device, self.gi = wl, c, torch.device(device), gi
        dt = c.dtype
        tdt = torch.float32 if dt == "f32" else torch.bfloat16
        dev = self.device
        cold, emb, hk, hv = growth_arrays(wl, gi)
        self.hot_pool = torch.zeros((c.hot_pages, 2, c.C, c.D), dtype=tdt, device=dev)
        self.W_q = to_torch(wl.W_q, dt).to(dev)
        self.cold = [to_torch(x, dt).pin_memory() for x in cold]
        self.emb = [to_torch(x, dt).to(dev) for x in emb]
        self.hca_k = [to_torch(x, dt).to(dev) for x in hk]
        self.hca_v = [to_torch(x, dt).to(dev) for x in hv]
        self.win_k = [to_torch(x, dt).to(dev) for x in wl.win_k]
        self.win_v = [to_torch(x, dt).to(dev) for x in wl.win_v]
        seqs = []
        for b in range(c.B):
            seqs.append(dict(cold_csa=self.cold[b], n_csa=c.n_csa(b), chunk_emb=self.emb[b], hca_k=self.hca_k[b], hca_v=self.hca_v[b],
                             n_hca=c.n_hca(b), win_k=self.win_k[b], win_v=self.win_v[b], w_len=min(c.W, c.L[b]),
                             w_head=min(c.W, c.L[b]) % c.W, step0=c.step0(b), cap_csa=gi.cap_csa(b), cap_hca=gi.cap_hca(b)))
        kw = dict(dtype=lsa.LSA_F32 if dt == "f32" else lsa.LSA_BF16, H=c.H, D=c.D, C_=c.C, W=c.W, Dh=c.Dh, E=c.E,
                  k=c.k, tau=c.tau, hot_pool=self.hot_pool, W_q=self.W_q, seqs=seqs, recall_lag=c.recall_lag)
        kw.update(ctx_over)
        self.ctx = lsa.LsaContext(**kw)
        self.tdt = tdt


def run_growth_lockstep(wl: LsaWorkload, gi, rig: "GrowthRig", steps: int, check_attention_at=None, check_tables_every: int = 1):
    """lsa_append_compressed + lsa_step against GrowingLsaOracle: the recalled part of every staged table is validated
    against the oracle's scores and fed back (tolerance cascade), then tables (recalled + tier entries), residency, counters,
    fetched bytes, exported cold-pool bytes and the tier pages' valid rows are compared bit for bit, attention within tolerance."""
    import torch
    from oracle import validate_selection
    from paper_2606_09079_b200.workloads import from_torch
    c = wl.cfg
    orc = make_growing_oracle(wl, gi)
    tol = attn_tolerance(c.dtype)
    n_checked, max_err, n_recalled_grown = 0, 0.0, 0
    ids = list(range(c.B))
    for t in range(steps):
        # ---- hand over what is due before step t (R29), both sides ----
        hca = gi.hca_entry(t) if gi.hca_due(t) else None
        csa = gi.csa_entry(t) if gi.csa_due(t) else None
        if hca is not None or csa is not None:
            emb_rows = None
            if csa is not None:
                rows = np.zeros((c.B, c.E), dtype=wl.W_q.dtype)
                need = False
                for b in range(c.B):
                    if orc.n_csa[b] % c.C == c.C - 1:
                        rows[b] = gi.emb_row(b, orc.n_csa[b] // c.C)
                        need = True
                emb_rows = rig.dev(rows) if need else None
            rig.ctx.append_compressed(ids, None if csa is None else rig.dev(csa[0]), None if csa is None else rig.dev(csa[1]),
                                      None if hca is None else rig.dev(hca[0]), None if hca is None else rig.dev(hca[1]), emb_rows)
            done = oracle_appends(orc, gi, t)
            if done:
                rig.ctx.sync()
                for b, ch in done:                                  # export: the cold pool's copy, bit for bit
                    got = from_torch(rig.cold[b][ch], c.dtype)
                    assert np.array_equal(got, orc.cold[b][ch]), f"step {t} seq {b}: exported chunk {ch} differs"
                    got_e = from_torch(rig.emb[b][ch].cpu(), c.dtype)
                    assert np.array_equal(got_e, orc.chunk_emb[b][ch]), f"step {t} seq {b}: embedding row {ch}"
        q, h = wl.q(t), wl.h(t)
        kn, vn = wl.kv_new(t)
        firing = [b for b in range(c.B) if orc.step[b] % c.tau == 0]
        out_gpu = rig.ctx.step(rig.dev(q), rig.dev(h), rig.dev(kn), rig.dev(vn))
        which = 0 if c.recall_lag == 0 else 1
        forced = {}
        for b in firing:
            chunks, pages = rig.ctx.page_table(b, which)
            rec = [ch for ch, p in zip(chunks, pages) if p < orc.P_lru]
            sc = orc.scores(b, h[b])
            order = sorted(rec, key=lambda ch: (-sc[ch], ch))
            padded = np.full(orc.k_sel, -1, dtype=np.int64); padded[: len(order)] = order
            msg = validate_selection(padded, sc, orc.k_sel)
            assert msg is None, f"step {t} seq {b}: {msg}"
            forced[b] = rec
        orc.step_begin(h, forced_selection=forced if firing else None)
        for b in firing:
            chunks, pages = rig.ctx.page_table(b, which)
            assert list(zip(chunks, pages)) == orc.table(b, which), f"step {t} seq {b}: staged table {list(zip(chunks, pages))} vs {orc.table(b, which)}"
            n = orc.n_chunks[b]
            assert rig.ctx.residency(b, n) == orc.pool.page_of[b][:n], f"step {t} seq {b}: residency mismatch"
            n_recalled_grown += sum(1 for ch in forced[b] if ch >= c.n_csa(b) // c.C)
        if firing:
            st = rig.ctx.stats()
            assert (st["hits"], st["misses"], st["evictions"], st["bytes_fetched"], st["pool_error"], st["chunks_exported"]) == \
                   (orc.pool.hits, orc.pool.misses, orc.pool.evictions, orc.pool.bytes_fetched, 0, orc.exported), f"step {t}: counters"
            hot_np = from_torch(rig.hot_pool.cpu(), c.dtype)
            owned = [p for p, o in enumerate(orc.pool.owner) if o is not None]
            assert np.array_equal(hot_np[owned], orc.pool.hot[owned]), f"step {t}: fetched bytes differ"
        if t % check_tables_every == 0:
            for b in range(c.B):
                chunks, pages = rig.ctx.page_table(b, 0)
                assert list(zip(chunks, pages)) == orc.table(b, 0), f"step {t} seq {b}: current table {list(zip(chunks, pages))} vs {orc.table(b, 0)}"
            hot_np = from_torch(rig.hot_pool.cpu(), c.dtype)
            for b in range(c.B):
                for ch in orc.tier(b):                             # the tier pages' valid rows
                    p, v = orc.tier_page(b, ch), orc.valid_rows(b, ch)
                    assert np.array_equal(hot_np[p][:, :v], orc.pool.hot[p][:, :v]), f"step {t} seq {b}: tier chunk {ch}"
        attend = check_attention_at is None or t in check_attention_at
        res = orc.step_end(q, kn, vn, attend=attend)
        if attend:
            got = rig.host(out_gpu)
            np.testing.assert_allclose(got, res[0], err_msg=f"attention mismatch at step {t}", **tol)
            max_err = max(max_err, float(np.max(np.abs(got - res[0]))))
            n_checked += 1
    rig.ctx.sync()
    st = rig.ctx.stats()
    for b in range(c.B):
        hk = from_torch(rig.hca_k[b].cpu(), c.dtype)
        assert np.array_equal(hk[: orc.n_hca[b]], orc.hca_k[b][: orc.n_hca[b]])
    return dict(checked=n_checked, max_abs_err=max_err, oracle=orc, exported=st["chunks_exported"], csa_appended=st["csa_appended"],
                hca_appended=st["hca_appended"], recalled_grown=n_recalled_grown)


# ------------------------------------------------------------------------------------------
# FP8 (e4m3) cold pages: the cold pool holds codes + block scales, a recall dequantises (DESIGN R34)
# ------------------------------------------------------------------------------------------
def make_fp8_oracle(wl: LsaWorkload, fp8, **over) -> LsaOracle:
    """The oracle of a run whose cold pool is `fp8` (workloads.Fp8ColdInputs): its cold pages are what a recall must write
    into the hot pool - the codes dequantised by oracle/fp8_oracle.py - and a page costs C*D*2 bytes on the host link."""
    from oracle.fp8_oracle import dequant_page
    c = wl.cfg
    cold = []
    for b in range(c.B):
        pages = np.empty(fp8.codes[b].shape, dtype=np.uint16)
        for ch in range(pages.shape[0]):
            pages[ch] = dequant_page(fp8.codes[b][ch], fp8.scales[b][ch])
        cold.append(pages)
    return make_oracle(wl, cold_csa=cold, cold_page_nbytes=2 * c.C * c.D, **over)


class Fp8Rig(GpuRig):
    """GpuRig with lsa_config.cold_format = FP8_E4M3: pinned uint8 code pools, device scale arrays."""

    def __init__(self, wl: LsaWorkload, fp8, device="cuda:0", **ctx_over):
        import torch
        from paper_2606_09079_b200 import lsa
        from paper_2606_09079_b200.workloads import to_torch
        c = wl.cfg
        assert c.dtype == "bf16"
        self.wl, self.cfg, self.device, self.fp8 = wl, c, torch.device(device), fp8
        dev, tdt = self.device, torch.bfloat16
        self.hot_pool = torch.zeros((c.hot_pages, 2, c.C, c.D), dtype=tdt, device=dev)
        self.W_q = to_torch(wl.W_q, "bf16").to(dev)
        self.cold = [torch.from_numpy(x.copy()).pin_memory() for x in fp8.codes]
        self.cold_scale = [torch.from_numpy(x.copy()).to(dev) for x in fp8.scales]
        self.emb = [to_torch(wl.chunk_emb(b, 0), "bf16").to(dev) for b in range(c.B)]
        self.hca_k = [to_torch(x, "bf16").to(dev) for x in wl.hca_k]
        self.hca_v = [to_torch(x, "bf16").to(dev) for x in wl.hca_v]
        self.win_k = [to_torch(x, "bf16").to(dev) for x in wl.win_k]
        self.win_v = [to_torch(x, "bf16").to(dev) for x in wl.win_v]
        seqs = [dict(cold_csa=self.cold[b], cold_scale=self.cold_scale[b], n_csa=c.n_csa(b), chunk_emb=self.emb[b], hca_k=self.hca_k[b],
                     hca_v=self.hca_v[b], win_k=self.win_k[b], win_v=self.win_v[b], w_len=min(c.W, c.L[b]),
                     w_head=min(c.W, c.L[b]) % c.W, step0=c.step0(b)) for b in range(c.B)]
        kw = dict(dtype=lsa.LSA_BF16, H=c.H, D=c.D, C_=c.C, W=c.W, Dh=c.Dh, E=c.E, k=c.k, tau=c.tau, hot_pool=self.hot_pool,
                  W_q=self.W_q, seqs=seqs, recall_lag=c.recall_lag, cold_format=lsa.LSA_COLD_FP8_E4M3)
        kw.update(ctx_over)
        self.ctx = lsa.LsaContext(**kw)
        self.tdt = tdt
