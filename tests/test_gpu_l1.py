"""Parity of the paper-exact Level-1 Memory Indexer (lsa_l1_init / lsa_l1_select; Eq.(1)-(5), (13))
against oracle/l1_oracle.py on the same seeded inputs.

The GPU matches entries on bf16 tensor cores with the query kept as TWO bf16 terms (hi + lo, fp32 accumulation of
both products); the oracle is fp64 from the stored inputs.  Per query element that leaves a relative error of 2^-17
instead of 2^-9, a pre-activation error below 1e-3 at magnitudes up to ~20, and dI <= dpre / 4: the chunk score
I = sigmoid(pre) is compared with atol 2e-3 and the selection with validate_l1_selection's band of 2e-3 around the
threshold / the K_max cut-off (3e-2 with a single bf16 term).  Everything integer downstream
(page tables after lsa_fetch_chunks) is checked exactly against the GPU's own selection."""
import numpy as np
import pytest
import torch

from lsa_harness import GpuRig, run_lockstep
from oracle.l1_oracle import l1_index_select, validate_l1_selection
from paper_2606_09079_b200.workloads import L1Inputs, LsaWorkload, make_small_config, to_torch

pytestmark = pytest.mark.gpu
BAND = 2e-3


def _rig(cfg, n_layers, d_c):
    wl = LsaWorkload(cfg)
    l1 = L1Inputs(wl, n_layers=n_layers, d_c=d_c)
    rig = GpuRig(wl)
    dev = rig.device
    layers = [{k: to_torch(v, "bf16").to(dev) for k, v in lay.items()} for lay in l1.layers]
    index_k = [[to_torch(K, "bf16").to(dev) for K in l1.index_k[b]] for b in range(cfg.B)]
    rig.ctx.l1_init(layers, index_k, d_c=d_c)
    return wl, l1, rig


@pytest.mark.parametrize("k,n_layers", [(12, 3), (40, 3), (3, 1)])
def test_l1_select_matches_oracle(k, n_layers):
    cfg = make_small_config("bf16", B=3, L=[20096, 4992, 512], C=128, H=8, D=64, Dh=512, E=64, k=k, hot_pages=2 * (min(k, 40) + min(k, 10) + 1) + 8,
                            W=64)
    wl, l1, rig = _rig(cfg, n_layers, 128)
    for t in (0, 3):
        h = wl.h(t)
        sel, sc = rig.ctx.l1_select(rig.dev(h), [0, 1, 2])
        rig.ctx.sync()
        sel, sc = sel.cpu().numpy(), sc.cpu().numpy().astype(np.float64)
        for b in range(cfg.B):
            o_sel, o_val, cs, _ = l1_index_select(h[b], l1.layers, l1.index_k[b], 64, cfg.C, k)
            msg = validate_l1_selection(sel[b], cs, k, 0.5, BAND)
            assert msg is None, f"step {t} seq {b}: {msg}\n gpu {sel[b]}\n oracle {o_sel}"
            valid = sel[b] >= 0
            np.testing.assert_allclose(sc[b][valid], cs[sel[b][valid]], atol=BAND)
            assert np.all(sc[b][~valid] == -np.inf)
            got = sc[b][valid]
            assert np.all(got[:-1] >= got[1:]), "scores must come out in non-increasing order"
    # subset call: rows of h follow seq_ids
    h = wl.h(5)
    sel2, _ = rig.ctx.l1_select(rig.dev(h[[0, 2]]), [0, 2])
    sel_all, _ = rig.ctx.l1_select(rig.dev(h), [0, 1, 2])
    rig.ctx.sync()
    assert torch.equal(sel2[0], sel_all[0]) and torch.equal(sel2[1], sel_all[2])
    # the selection feeds S4-S5 unchanged
    rig.ctx.fetch_chunks([0, 1, 2], sel_all)
    rig.ctx.commit_tables()
    for b in range(cfg.B):
        chunks, pages = rig.ctx.page_table(b)
        assert chunks == sorted(c for c in sel_all[b].cpu().tolist() if c >= 0)
        hot = rig.hot_pool.cpu()
        for c_, p_ in zip(chunks, pages):
            assert torch.equal(hot[p_], rig.cold[b][c_])
    rig.ctx.close()


def test_l1_select_at_the_bench_shape():
    """The shape `bench.py --l1` times: Dh = 4096, d_c = 2048 (the paper's r), 3 layers - rows of 4096 / 2048 weights take
    the multi-batch, double-buffered path of l1_gemv_kernel (a batch is 2048 weights) - and 65 536 compressed entries
    (512 chunks) per layer.  Chunk scores element by element and the selection against the oracle."""
    from paper_2606_09079_b200.workloads import make_config
    cfg = make_config(3, L=[262144], W=1024, hot_pages=160, steps=4, name="cfg3_quarter_l1")
    assert cfg.Dh == 4096 and cfg.n_csa(0) == 65536 and cfg.k == 64
    wl, l1, rig = _rig(cfg, 3, 2048)
    for t in (0, 1):
        h = wl.h(t)
        sel, sc = rig.ctx.l1_select(rig.dev(h), [0])
        rig.ctx.sync()
        sel, sc = sel.cpu().numpy(), sc.cpu().numpy().astype(np.float64)
        o_sel, o_val, cs, _ = l1_index_select(h[0], l1.layers, l1.index_k[0], 64, cfg.C, cfg.k)
        msg = validate_l1_selection(sel[0], cs, cfg.k, 0.5, BAND)
        assert msg is None, f"step {t}: {msg}\n gpu {sel[0]}\n oracle {o_sel}"
        valid = sel[0] >= 0
        assert valid.sum() >= 8, "the planted structure should recall chunks"
        np.testing.assert_allclose(sc[0][valid], cs[sel[0][valid]], atol=BAND)
    rig.ctx.close()


def test_lsa_step_with_level1_indexer_lockstep():
    """lsa_set_indexer(LEVEL1): the paper-exact indexer drives lsa_step (trigger -> Eq.1-5,13 -> residency ->
    fetch -> attention).  The GPU's selection is validated against the L1 oracle, then page tables, residency,
    counters, fetched bytes (bit-exact) and attention outputs (BASELINE tolerance) are checked in lock-step."""
    from paper_2606_09079_b200 import lsa
    cfg = make_small_config("bf16", B=3, L=[20096, 4992, 512], C=128, H=8, D=64, Dh=512, E=64, k=10, hot_pages=64, W=64, tau=4, steps=14)
    wl, l1, rig = _rig(cfg, 2, 128)
    rig.ctx.set_indexer(lsa.LSA_INDEXER_LEVEL1)
    r = run_lockstep(wl, rig, cfg.steps, l1=l1, l1_band=BAND)
    assert r["checked"] == cfg.steps
    st = rig.ctx.stats()
    assert st["misses"] > 0 and st["hits"] > 0            # h drifts slowly: later triggers mostly hit
    rig.ctx.close()


def test_l1_rejects_unsupported_shapes():
    from paper_2606_09079_b200 import lsa
    cfg = make_small_config("bf16", B=1, L=[4096], C=16, H=8, D=64, Dh=128, E=64, k=3, hot_pages=16, W=64)
    wl = LsaWorkload(cfg)
    rig = GpuRig(wl)
    z = torch.zeros((64, 128), dtype=torch.bfloat16, device=rig.device)
    with pytest.raises(lsa.LsaError) as e:
        rig.ctx.l1_init([dict(W_dq=z, W_iuq=z, W_w=z)], [[z]], d_c=64)      # C = 16: no kernel
    assert e.value.code == -6
    with pytest.raises(lsa.LsaError):
        rig.ctx.l1_select(z, [0])                                          # not initialised
    rig.ctx.close()
