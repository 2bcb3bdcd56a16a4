"""FP8 (e4m3) cold pages: S5 dequantises while it copies, lsa_export_chunks quantises (R34-R36).  GPU parity
against oracle/fp8_oracle.py + the lock-step oracle: recalled hot pages, tables, residency, counters (bytes = HALF a hot
page per miss) bit for bit; attention within the bf16 tolerance."""
import numpy as np
import pytest
import torch

from lsa_harness import Fp8Rig, GpuRig, make_fp8_oracle, run_lockstep
from paper_2606_09079_b200.workloads import Fp8ColdInputs, LsaWorkload, from_torch, make_config, make_small_config, to_torch


def _cfg(**kw):
    base = dict(B=2, L=[32768 + 512, 16384], H=64, D=512, C=128, W=512, Dh=256, E=128, k=6, tau=8, steps=0, hot_pages=24,
                needle_period=2, n_needles=3)
    base.update(kw)
    return make_small_config("bf16", **base)


@pytest.mark.gpu
@pytest.mark.parametrize("overlap", [0, 1])
def test_fp8_cold_pool_lockstep_tcgen05(overlap):
    """BASELINE shape (H 64, D 512, C 128), needles drifting every 2 triggers so that pages are recalled throughout, a small
    pool so that pages are evicted and recalled again; one sequence ends in a partial chunk."""
    wl = LsaWorkload(_cfg())
    fp8 = Fp8ColdInputs(wl)
    rig = Fp8Rig(wl, fp8, step_overlap=overlap)
    res = run_lockstep(wl, rig, 72, check_attention_at=set(range(0, 72, 5)) | {1, 9, 17}, oracle=make_fp8_oracle(wl, fp8))
    st = rig.ctx.stats()
    assert st["misses"] > 12 and st["evictions"] > 0
    assert st["bytes_fetched"] == st["misses"] * wl.cfg.C * wl.cfg.D * 2          # one byte per element crossed the link
    assert res["checked"] >= 15


@pytest.mark.gpu
def test_fp8_cold_pool_churn_shape_shared_pool():
    """cfg 5's structure scaled down (uniform embeddings, h redrawn at every trigger, tau = 4): nearly every selected chunk is a
    miss, the shared pool is full after two triggers."""
    wl = LsaWorkload(_cfg(B=3, L=[16384, 16384, 8192 + 256], k=8, tau=4, hot_pages=2 * 8 * 3, emb_mode="uniform", n_needles=0,
                          kv_base_chunks=16))
    fp8 = Fp8ColdInputs(wl)
    rig = Fp8Rig(wl, fp8)
    run_lockstep(wl, rig, 40, check_attention_at={0, 1, 5, 21, 39}, oracle=make_fp8_oracle(wl, fp8))
    st = rig.ctx.stats()
    assert st["misses"] > 100 and st["evictions"] > 50


@pytest.mark.gpu
def test_fp8_export_quantises_like_the_oracle_and_round_trips_through_a_recall():
    """lsa_export_chunks with FP8 cold pages: codes and scales bit for bit against oracle.fp8_oracle.quantize_page on bf16
    pages whose blocks differ in magnitude by orders (so the block exponent rule is exercised), then a recall of those chunks
    must leave dequant(quant(page)) in the hot pool."""
    from oracle.fp8_oracle import dequant_page, quantize_page
    from paper_2606_09079_b200 import lsa
    wl = LsaWorkload(_cfg())
    c = wl.cfg
    fp8 = Fp8ColdInputs(wl)
    rig = Fp8Rig(wl, fp8)
    g = np.random.default_rng(77)
    n = 5
    pages = g.standard_normal((n, 2, c.C, c.D)).astype(np.float32)
    pages[0, 0] *= 3.0e-3; pages[1, 1] *= 40.0; pages[2] *= 1.0 / np.sqrt(c.D); pages[3, 0] = 0.0; pages[4, 1, 5:] = 0.0
    pages[2, 0, 0, :8] = [1.0625, 1.1875, -1.0625, 2.0 ** -12, 0.0, -0.0, 0.124, 0.126]       # ties and tiny values
    src = torch.from_numpy(pages).to(torch.bfloat16).cuda()
    rig.ctx.export_chunks(1, 3, src)
    rig.ctx.sync()
    wide = src.to(torch.float32).cpu().numpy()
    for i in range(n):
        codes, scales = quantize_page(wide[i])
        got = rig.cold[1][3 + i].numpy()
        assert np.array_equal(got, codes), f"page {i}: {np.argwhere(got != codes)[:4]}"
        assert np.array_equal(rig.cold_scale[1][3 + i].cpu().numpy(), np.array(scales, dtype=np.float32))
    # neighbours untouched
    assert np.array_equal(rig.cold[1][2].numpy(), fp8.codes[1][2]) and np.array_equal(rig.cold[1][8].numpy(), fp8.codes[1][8])
    # recall the exported chunks explicitly and look at the hot pool
    sel = torch.full((1, c.k), -1, dtype=torch.int32, device="cuda")
    sel[0, :n] = torch.arange(3, 3 + n, dtype=torch.int32)
    rig.ctx.fetch_chunks([1], sel)
    rig.ctx.commit_tables()
    rig.ctx.sync()
    chunks, pgs = rig.ctx.page_table(1, 0)
    assert chunks == list(range(3, 3 + n))
    hot = from_torch(rig.hot_pool.cpu(), "bf16")
    for ch, p in zip(chunks, pgs):
        codes, scales = quantize_page(wide[ch - 3])
        assert np.array_equal(hot[p], dequant_page(codes, scales)), f"chunk {ch}"
    # the error a page suffers on its way through the cold pool: half an ulp of a 3-bit mantissa, relative to the block maximum
    back = (hot[pgs[2]].astype(np.uint32) << 16).view(np.float32)
    assert np.max(np.abs(back - wide[2])) <= np.max(np.abs(wide[2])) * 2.0 ** -4


@pytest.mark.gpu
def test_fp8_cold_pool_argument_errors():
    from paper_2606_09079_b200 import lsa
    wl = LsaWorkload(_cfg())
    fp8 = Fp8ColdInputs(wl)
    good = Fp8Rig(wl, fp8)
    with pytest.raises(lsa.LsaError):                        # scales missing
        seqs = [dict(cold_csa=good.cold[b], n_csa=wl.cfg.n_csa(b), chunk_emb=good.emb[b], hca_k=good.hca_k[b], hca_v=good.hca_v[b],
                     win_k=good.win_k[b], win_v=good.win_v[b], w_len=512, w_head=0) for b in range(2)]
        lsa.LsaContext(dtype=lsa.LSA_BF16, H=64, D=512, C_=128, W=512, Dh=256, E=128, k=6, tau=8, hot_pool=good.hot_pool, W_q=good.W_q,
                       seqs=seqs, cold_format=lsa.LSA_COLD_FP8_E4M3)
    wl32 = LsaWorkload(make_small_config("f32"))
    with pytest.raises(lsa.LsaError):                        # fp32 hot pages cannot take FP8 cold pages
        GpuRig(wl32, cold_format=lsa.LSA_COLD_FP8_E4M3)
