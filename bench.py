#!/usr/bin/env python
"""bench.py - LSA decode-step throughput on B200 through the C ABI (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one pass of the whole hot path (lsa_step: table swap, window append, split-K attention
+ merge, and - every tau steps - query tower, chunk scoring, top-k, residency diff, chunk fetch on
the side stream) over one decode token of every sequence of the config.  Default workload =
BASELINE.json configs[2] (1-based config 3: bf16, B=1, 1M-token context), the one the metric is
quoted on.  Inputs are synthetic and seeded (paper_2606_09079_b200/workloads.py).

L2 hygiene: the per-step working set at B=1 (48 MiB) fits B200's L2, so R independent replicas of the
layer state are stepped round-robin with R * bytes/step >= 2x L2 ("inputs larger than L2"); a real
model touches >= 21 such layers per token.  The replicas start at trigger phases
spread over tau and the warm-up covers every replica's first (cold) trigger, so that any timed window,
however short, holds steady-state triggers: replica 0 fires at the first timed step.

The steps of the timed loop are independent of one another (different replicas, inputs staged before
the loop), so the contexts are created with lsa_config.step_overlap = 1 (--overlap 0 for the default
of the API, where q / k_new / v_new may be produced by the work enqueued just before the call); the
line carries the other mode as `dependent_inputs`.

`--gpus N` (N > 1) without a torchrun environment re-executes this file under torch.distributed.run,
one rank per GPU: configs 4 and 5 shard their sequences over the ranks (strong scaling: each GPU brings
its own host link), the single-sequence configs run one replica set per rank (weak scaling); no
data-path collective either way.  `--dry-run` drives that launcher and the reductions on CPU (gloo).

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload; the oracle is otherwise only used for the `cpu_baseline` leg on rank 0.
"""
import argparse
import hashlib
import json
import math
import os
import socket
import subprocess
import sys
import threading
import time
import types

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_09079_b200.dist import max_over_ranks, shard_sequences, sum_over_ranks  # noqa: E402
from paper_2606_09079_b200.workloads import Fp8ColdInputs, LsaWorkload, make_config, plant_boundary_ties, shard_config, to_torch  # noqa: E402

METRIC = {1: ("lsa_decode_steps_per_s_8k_ctx_fp32", "steps/s"),
          2: ("lsa_decode_steps_per_s_128k_ctx", "steps/s"),
          3: ("lsa_decode_steps_per_s_1m_ctx", "steps/s"),
          4: ("lsa_decode_tokens_per_s_b32_ragged", "tokens/s"),
          5: ("lsa_decode_steps_per_s_churn_b8_512k", "steps/s")}
SHARDED = (4, 5)                 # configs whose sequences are spread over the ranks (strong scaling)
L2_DEFAULT = 126 * 2**20


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d["hbm_gbs"], source="MEASURED_PEAKS.json (of measured)")
    return dict(hbm_gbs=6650.0, source="B200_PROFILING.md fallback (of fallback)")


def kernel_source_digest():
    """sha-256 prefix of the sources of the dominant kernel: a stored ncu figure is only quoted while it still
    describes the code that runs (profiles/r02_traffic.txt)."""
    h = hashlib.sha256()
    for f in ("lsa_attn_tc_small.cuh", "lsa_attn_tc_kernel.cuh", "lsa_attn_tc_defs.cuh", "lsa_tc_ptx.cuh"):
        h.update(open(os.path.join(ROOT, "paper_2606_09079_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:16]


def stored_traffic(config_id, overlap):
    """dram__bytes_read + dram__bytes_write of one launch of the dominant kernel from the committed ncu --set full capture
    (profiles/), or None when there is no capture for this config or the kernel sources have changed since."""
    p = os.path.join(ROOT, "profiles", "r02_traffic.txt")
    if not os.path.exists(p):
        return None, "no capture"
    d = json.load(open(p)).get(f"cfg{config_id}_overlap{overlap}")
    if not d:
        return None, "no capture for this config"
    if d.get("source_sha16") != kernel_source_digest():
        return None, f"capture of commit {d.get('commit')} is stale: kernel sources changed"
    return d["traffic_bytes"], f"ncu --set full, commit {d.get('commit')} ({d.get('file')})"


def summarise_timeline(records, step_ms):
    """Per-CTA timeline of the small-batch attention launches (include/lsa.h LSA_TL_*): records = one uint64 array
    [launch record][CTA][event] per context.  Means over all stamped CTAs, in microseconds: where a CTA's residence on its SM
    goes, how long an SM stays empty between two CTAs, and the step time that SM residence alone would give."""
    import numpy as np
    ENTRY, SETUP, FIRST_S, LAST_PV, EPI, ARRIVED, ALL_ARR, MERGED, EXIT, SMID, NCTAS, SEQ = range(12)
    rows = []
    n_launches = 0
    for rec in records:
        a = rec.astype(np.int64)
        for l in range(a.shape[0]):
            n = int(a[l, 0, NCTAS])
            if n <= 0 or n > a.shape[1] or (a[l, :n, EXIT] <= a[l, :n, ENTRY]).any():
                continue                            # never written, or overwritten while it was read
            rows.append(a[l, :n])
            n_launches += 1
    if not rows:
        return None
    e = np.concatenate(rows)
    mrg = e[:, MERGED] > 0
    us = lambda x: float(np.mean(x)) / 1e3
    res = e[:, EXIT] - e[:, ENTRY]
    by_sm = {}
    for r_ in e:
        by_sm.setdefault(int(r_[SMID]), []).append((int(r_[ENTRY]), int(r_[EXIT])))
    gaps = []
    for v in by_sm.values():
        v.sort()
        gaps += [b0 - a1 for (_, a1), (b0, _) in zip(v, v[1:]) if 0 <= b0 - a1 < 8000]     # consecutive CTAs on one SM
    sm_us_per_launch = float(res.sum()) / 1e3 / n_launches
    handover = float(np.median(gaps)) / 1e3 if gaps else None
    ctas = len(e) / n_launches
    out = dict(launches=n_launches, ctas_per_launch=ctas, mergers_per_launch=float(mrg.sum()) / n_launches, sms_seen=len(by_sm),
               step_us=step_ms * 1e3,
               all_ctas_us=dict(entry_to_setup=us(e[:, SETUP] - e[:, ENTRY]), entry_to_first_s=us(e[:, FIRST_S] - e[:, ENTRY]),
                                first_s_to_last_pv=us(e[:, LAST_PV] - e[:, FIRST_S]), last_pv_to_epilogue=us(e[:, EPI] - e[:, LAST_PV]),
                                epilogue_to_arrived=us(e[:, ARRIVED] - e[:, EPI])),
               leavers_us=dict(residence=us(res[~mrg])) if (~mrg).any() else None,
               mergers_us=dict(arrived_to_all_arrived=us(e[mrg, ALL_ARR] - e[mrg, ARRIVED]), all_arrived_to_merged=us(e[mrg, MERGED] - e[mrg, ALL_ARR]),
                               residence=us(res[mrg])),
               sm_residence_us_per_launch=sm_us_per_launch, handover_us_median=handover,
               step_us_if_sm_bound=(sm_us_per_launch + ctas * (handover or 0.0)) / 148.0,
               note="stamps of %globaltimer by one thread per CTA; step_us is the step time of the stamped stretch (the stamps cost a little); "
                    "step_us_if_sm_bound = (summed residence + hand-over per CTA) / 148 SMs")
    return out


def replicas_for(c, l2_bytes):
    return max(1, math.ceil(2 * l2_bytes / c.attn_bytes_per_step()))


def workload_config(c, n_gpus, l2_bytes=L2_DEFAULT):
    """The `config` object of the JSON line: the workload only, identical for both arms."""
    R = replicas_for(c, l2_bytes)
    B = c.B_total or c.B
    return dict(workload=c.name, B=B, L=c.L if B <= 2 else f"{min(c.L)}..{max(c.L)}", H=c.H, D=c.D,
                C=c.C, W=c.W, Dh=c.Dh, E=c.E, k=c.k, tau=c.tau, hot_pages=c.hot_pages, recall_lag=c.recall_lag,
                cold_pool=("tiled from %d seeded base chunks, one tagged element per chunk" % c.kv_base_chunks) if c.kv_base_chunks else "independent seeded streams",
                tie_triggers=c.tie_frac,
                l2_policy=f"{R} layer-state replicas stepped round-robin; {R}x{c.attn_bytes_per_step() / 2**20:.1f} MiB attended "
                          f"per rotation vs L2 {l2_bytes / 2**20:.0f} MiB (inputs larger than L2)",
                parallelism=f"dp{n_gpus} (" + ("sequences sharded over ranks" if c.config_id in SHARDED and n_gpus > 1 else "independent sequences per rank") + ", no collective)")


# ----------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the oracle on a bounded sample
# ----------------------------------------------------------------------------------------------
def oracle_sample(wl, budget_s=20.0, max_steps=24, threads=None):
    """Run the oracle as it stands from step 0 (trigger + fetch + attention) for up to max_steps steps
    or ~budget_s seconds; returns (steps, seconds, threads)."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from lsa_harness import make_oracle
    from threadpoolctl import threadpool_info, threadpool_limits
    used = os.cpu_count() or 1
    nt = [i.get("num_threads", 1) for i in threadpool_info() if i.get("user_api") == "blas"]
    if nt:
        used = max(nt)

    def run():
        orc = make_oracle(wl)
        t0 = time.perf_counter()
        n = 0
        while n < max_steps:
            kn, vn = wl.kv_new(n)
            orc.run_step(wl.q(n), wl.h(n), kn, vn)
            n += 1
            if time.perf_counter() - t0 > budget_s:
                break
        return n, time.perf_counter() - t0

    if threads is None:
        n, secs = run()
        return n, secs, used
    with threadpool_limits(limits=threads):
        n, secs = run()
    return n, secs, threads


def run_reference(args, cfg, wl):
    name, unit = METRIC[cfg.config_id]
    per_step_units = cfg.B if unit == "tokens/s" else 1
    for _ in range(max(args.warmup, 0) and 1):
        oracle_sample(wl, budget_s=1.0, max_steps=1)
    n, secs, threads = oracle_sample(wl, budget_s=max(5.0, min(60.0, 2.0 * args.steps)), max_steps=max(2, min(args.steps, 48)))
    val = n * per_step_units / secs
    line = dict(metric=name, value=val, unit=unit, n_gpus=args.gpus, steps=n, warmup=1, ms_per_step=1e3 * secs / n,
                higher_is_better=True, scaling="strong" if cfg.config_id in SHARDED and args.gpus > 1 else "weak", vs_baseline=None,
                dtype="f64", data="synthetic", impl="reference", config=workload_config(cfg, args.gpus),
                cpu_baseline=dict(value=val, unit=unit, cores=threads, kind="oracle",
                                  sample=f"oracle steps 0..{n - 1} of {cfg.name} (trigger + fetch at step 0, attention every step)"),
                e2e=dict(value=val, unit=unit, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


# ----------------------------------------------------------------------------------------------
# clocks: NVML in-process, sampled over the whole GPU phase
# ----------------------------------------------------------------------------------------------
class ClockSampler:
    """SM clock / throttle reasons read through NVML from a thread every few milliseconds between start() and stop();
    `window` is the wall-clock span of the timed region, so that samples inside it can be told apart."""

    def __init__(self, dev_index, interval_s=0.004):
        self.samples, self.window, self.err = [], None, None
        self._stop = threading.Event()
        self.interval = interval_s
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[dev_index]) if vis and all(x.strip().isdigit() for x in vis.split(",")) else dev_index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_sm = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:                                   # no NVML: say so, never guess
            self.nv, self.err = None, repr(e)

    def _one(self):
        nv = self.nv
        sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
        try:
            rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            rs = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        self.samples.append((time.perf_counter(), sm, rs))

    def _run(self):
        while not self._stop.is_set():
            try:
                self._one()
            except Exception as e:
                self.err = repr(e)
                return
            self._stop.wait(self.interval)

    def start(self):
        if self.nv is not None:
            self.th = threading.Thread(target=self._run, daemon=True)
            self.th.start()

    def sample_now(self):
        if self.nv is not None:
            try:
                self._one()
            except Exception as e:
                self.err = repr(e)

    def stop(self):
        if self.nv is None:
            return dict(sm_mhz=None, sm_max_mhz=None, samples=0, reasons=[f"NVML unavailable: {self.err}"])
        self._stop.set()
        self.th.join(timeout=2)
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        sm = [s[1] for s in self.samples]
        reasons = sorted(n for n, bit in names.items() if any(s[2] & bit for s in self.samples))
        inside = [s[1] for s in self.samples if self.window and self.window[0] <= s[0] <= self.window[1] + 0.002]
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=float(self.max_sm), samples=len(sm),
                    samples_in_timed_region=len(inside), sm_mhz_in_timed_region=float(np.median(inside)) if inside else None,
                    reasons=reasons, how="NVML in-process, every 4 ms from the first warm-up step to the end of the end-to-end leg")


# ----------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------
class Replica:
    def __init__(self, wl, shared, sc, sf, lsa, phase, overlap):
        c = wl.cfg
        dev = shared["dev"]
        tdt = shared["tdt"]
        self.hot_pool = torch.zeros((c.hot_pages, 2, c.C, c.D), dtype=tdt, device=dev)
        self.emb = [e.clone() for e in shared["emb"]]
        self.hca_k = [x.clone() for x in shared["hca_k"]]
        self.hca_v = [x.clone() for x in shared["hca_v"]]
        self.win_k = [x.clone() for x in shared["win_k"]]
        self.win_v = [x.clone() for x in shared["win_v"]]
        fp8 = shared.get("cold_scale") is not None
        seqs = [dict(cold_csa=shared["cold"][b], cold_scale=shared["cold_scale"][b] if fp8 else None, n_csa=c.n_csa(b), chunk_emb=self.emb[b], hca_k=self.hca_k[b],
                     hca_v=self.hca_v[b], win_k=self.win_k[b], win_v=self.win_v[b], w_len=min(c.W, c.L[b]), w_head=0,
                     step0=c.step0(b) + phase) for b in range(c.B)]
        self.ctx = lsa.LsaContext(dtype=lsa.LSA_F32 if c.dtype == "f32" else lsa.LSA_BF16, H=c.H, D=c.D, C_=c.C, W=c.W,
                                  Dh=c.Dh, E=c.E, k=c.k, tau=c.tau, hot_pool=self.hot_pool, W_q=shared["W_q"], seqs=seqs,
                                  recall_lag=c.recall_lag, stream_compute=sc, stream_fetch=sf,
                                  attn_impl=shared["attn_impl"], max_ctas=shared.get("max_ctas", 0), step_overlap=overlap,
                                  cold_format=lsa.LSA_COLD_FP8_E4M3 if fp8 else lsa.LSA_COLD_NATIVE)
        self.step = phase                # global step index of the workload this replica is at (wl.fires / wl.trigger_index)
        self.bound = {}                  # lsa_step bound to fixed input buffers (LsaContext.bind_step)
        self.tie_emb = {}                # cfg 5: sequences whose alternate (tie-carrying) embedding table is installed


def relaunch_under_torchrun(args):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    env = dict(os.environ)
    if not args.dry_run:
        env.setdefault("NCCL_DEBUG", "INFO")          # the ranks show up in NCCL's own log (stderr)
    return subprocess.run(cmd, env=env).returncode


def dry_run(args, cfg, rank, world):
    """The N > 1 plumbing without a GPU: gloo group, sequence shards, the two reductions, one line from rank 0."""
    import torch.distributed as dist
    if world > 1:
        dist.init_process_group("gloo")
    sharded = cfg.config_id in SHARDED and world > 1
    lo, hi = shard_sequences(cfg.B, world, rank) if sharded else (0, cfg.B)
    sub = shard_config(cfg, lo, hi) if sharded else cfg
    name, unit = METRIC[cfg.config_id]
    tokens = unit == "tokens/s"
    units = args.steps * (sub.B if tokens else 1) if (tokens or not sharded) else (args.steps if rank == 0 else 0)
    job_ms = max_over_ranks(10.0 * (1 + rank))                       # pretend the last rank is the slow one
    total = sum_over_ranks(units)
    shards = [None] * world
    if world > 1:
        dist.all_gather_object(shards, (lo, hi, sub.hot_pages))
    else:
        shards = [(lo, hi, sub.hot_pages)]
    if rank == 0:
        print(json.dumps(dict(metric=name, value=total / (job_ms * 1e-3), unit=unit, n_gpus=world, steps=args.steps, warmup=args.warmup,
                              ms_per_step=job_ms / args.steps, higher_is_better=True, scaling="strong" if sharded else "weak",
                              vs_baseline=None, dtype=cfg.dtype, data="synthetic", dry_run=True, shards=shards,
                              config=workload_config(cfg, world))))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20000)
    ap.add_argument("--warmup", type=int, default=256)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--recall-lag", type=int, default=None, help="override the config's recall_lag (default 1 = the paper's t+1; up to tau-1)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--attn", default="auto", choices=["auto", "simt", "tcgen05"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--replicas", type=int, default=0)
    ap.add_argument("--max-ctas", type=int, default=0, help="cap on attention CTAs (0 = library default)")
    ap.add_argument("--overlap", type=int, default=1, help="lsa_config.step_overlap of the timed contexts: 1 = the steps' inputs do not depend on the previous step's output (true of this loop); 0 = the API default")
    ap.add_argument("--no-dependent", action="store_true", help="skip the second measurement in the other step_overlap mode")
    ap.add_argument("--dry-run", action="store_true", help="CPU only: launcher, sharding and reductions with a gloo group")
    ap.add_argument("--l1", action="store_true", help="also time the paper-exact Level-1 indexer (NEXT-1)")
    ap.add_argument("--export", action="store_true", help="also time lsa_export_chunks (NEXT-4: KV export HBM -> pinned cold pool)")
    ap.add_argument("--cold-fp8", action="store_true", help="FP8 (e4m3) cold pages: half the bytes per recall over the host link (not BASELINE's config: reported under run.cold_format)")
    ap.add_argument("--growth", action="store_true", help="also time the step with a growing compressed history (NEXT-4: lsa_append_compressed)")
    ap.add_argument("--timeline", action="store_true", help="also stamp a per-CTA timeline of the small-batch attention launches (lsa_timeline_*) over a separate stretch of steps and summarise it")
    ap.add_argument("--graph", action="store_true", help="also time lsa_step_graph (NEXT-3: the non-trigger step replayed from a CUDA graph)")
    ap.add_argument("--l2", action="store_true", help="also time the step with Level 2 (native Top-k inside the resident set, NEXT-2)")
    ap.add_argument("--l2-k2", type=int, default=2048, help="Level-2 Top-k (entries per sequence and step)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        return relaunch_under_torchrun(args)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    cfg = make_config(args.config) if args.recall_lag is None else make_config(args.config, recall_lag=args.recall_lag)
    if args.impl == "reference":
        if rank == 0:
            run_reference(args, cfg, LsaWorkload(cfg))
        return 0
    if args.dry_run:
        return dry_run(args, cfg, rank, world)

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    from paper_2606_09079_b200 import lsa

    sharded = cfg.config_id in SHARDED and world > 1
    if sharded:                                        # this rank's sequences only: own pools, own host link
        lo, hi = shard_sequences(cfg.B, world, rank)
        c = shard_config(cfg, lo, hi)
    else:
        c = cfg
    wl = LsaWorkload(c)
    tdt = torch.float32 if c.dtype == "f32" else torch.bfloat16
    name, unit = METRIC[c.config_id]
    tokens = unit == "tokens/s"
    per_step_units = c.B if tokens else 1
    props = torch.cuda.get_device_properties(dev)
    l2 = getattr(props, "L2_cache_size", L2_DEFAULT)
    attn_bytes = c.attn_bytes_per_step()
    R = args.replicas or replicas_for(c, l2)
    attn_impl = dict(auto=lsa.LSA_ATTN_AUTO, simt=lsa.LSA_ATTN_SIMT, tcgen05=lsa.LSA_ATTN_TCGEN05)[args.attn]

    def job_units(n_steps):
        """units of the whole job in n_steps steps: ranks with their own replica sets add up; ranks that share one
        batch of sequences make the same steps (tokens add up, steps do not)"""
        if sharded and not tokens:
            return n_steps
        return sum_over_ranks(n_steps * per_step_units, dev)

    fp8 = Fp8ColdInputs(wl) if args.cold_fp8 else None            # --cold-fp8: e4m3 codes + block scales in the cold pool
    shared = dict(dev=dev, tdt=tdt, attn_impl=attn_impl, max_ctas=args.max_ctas, W_q=to_torch(wl.W_q, c.dtype).to(dev),
                  cold=([torch.from_numpy(x).pin_memory() for x in fp8.codes] if fp8 else [to_torch(x, c.dtype).pin_memory() for x in wl.cold_csa]),
                  cold_scale=[torch.from_numpy(x).to(dev) for x in fp8.scales] if fp8 else None,
                  emb=[to_torch(wl.chunk_emb(b, 0), c.dtype).to(dev) for b in range(c.B)],
                  hca_k=[to_torch(x, c.dtype).to(dev) for x in wl.hca_k], hca_v=[to_torch(x, c.dtype).to(dev) for x in wl.hca_v],
                  win_k=[to_torch(x, c.dtype).to(dev) for x in wl.win_k], win_v=[to_torch(x, c.dtype).to(dev) for x in wl.win_v])
    sc, sf = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    # replica r starts r * (tau // R) steps before a trigger; replica 0 fires at its steps 0, tau, ...
    phases = [(c.tau - r * (c.tau // R)) % c.tau for r in range(R)]
    reps = [Replica(wl, shared, sc, sf, lsa, phases[r], args.overlap) for r in range(R)]
    # every replica's first (cold: empty hot pool) trigger and its table swap happen in the warm-up, which is a whole
    # number of trigger periods per replica: replica 0 then fires again at the first timed step
    warmup = max(args.warmup, 3, R * c.tau)
    warmup += (-warmup) % (R * c.tau)

    # a rotating set of per-step inputs, resident in HBM before the timed region
    NIN = 16
    qs = [to_torch(wl.q(i), c.dtype).to(dev) for i in range(NIN)]
    hs = [to_torch(wl.h(i * c.tau), c.dtype).to(dev) for i in range(NIN)]
    kns, vns = zip(*[(to_torch(a, c.dtype).to(dev), to_torch(b_, c.dtype).to(dev)) for a, b_ in (wl.kv_new(i) for i in range(NIN))])
    out = torch.empty((c.B, c.H, c.D), dtype=tdt, device=dev)
    # needle drift (cfg 2-4): rows to rewrite at each trigger index, staged on the device
    drift = {}
    max_trig = (2 * warmup + 6 * args.steps) // (c.tau * R) + 6
    for trig in range(1, max_trig + 1):
        for b in range(c.B):
            upd = wl.emb_row_updates(b, trig)
            if upd is not None:
                drift[(b, trig)] = (torch.from_numpy(upd[0]).to(dev), to_torch(upd[1], c.dtype).to(dev))
    # cfg 5 (BASELINE.json: "10% of triggers carry planted exact-tie and near-tie scores"): those triggers get an alternate
    # table with an exact tie across the k-th rank of a FIXED seeded ranking and a one-ulp near-tie behind it (the parity
    # tests plant them across the oracle's own ranking; here only the timing of the tie-break matters)
    tie_tables = {}
    if c.tie_frac > 0:
        for b in range(c.B):
            for trig in range(0, min(max_trig + 1, 256)):
                if wl.has_tie_trigger(b, trig) and len(tie_tables) < 32:
                    order = np.random.Generator(np.random.Philox(c.seed + 977 * b + trig)).permutation(c.n_chunks(b))
                    tie_tables[(b, trig)] = to_torch(plant_boundary_ties(wl.chunk_emb(b, trig), order, c.k_eff(b), c.dtype), c.dtype).to(dev)
    torch.cuda.synchronize()
    n_tie_triggers = [0]
    drift_needs_host_sync = False        # (the drift / tie updates of one_step are not replayed by the async leg: it keeps the tables)

    def one_step(i, host=None, rs=None):
        rs = reps if rs is None else rs
        r = rs[i % len(rs)]
        t = r.step
        if drift or tie_tables:
            for b in range(c.B):
                if not wl.fires(b, t):
                    continue
                trig = wl.trigger_index(b, t)
                u = drift.get((b, trig))
                if u is not None:
                    with torch.cuda.stream(sf):
                        r.emb[b][u[0]] = u[1]
                if (b, trig) in tie_tables:
                    r.ctx.set_chunk_emb(b, tie_tables[(b, trig)])
                    r.tie_emb[b] = True
                    n_tie_triggers[0] += 1
                elif r.tie_emb.get(b):
                    r.ctx.set_chunk_emb(b, r.emb[b])
                    r.tie_emb[b] = False
        j = i % NIN
        if host is None:
            key = (j, (t // c.tau) % NIN)
            fn = r.bound.get(key)
            if fn is None:
                fn = r.bound[key] = r.ctx.bind_step(qs[j], hs[key[1]], kns[j], vns[j], out)
            fn()
        else:
            r.ctx.step_host(host["q"][j], host["h"][(t // c.tau) % NIN], host["kn"][j], host["vn"][j], host["out"])
        r.step += 1

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    def counters(rs):
        st = [r.ctx.stats() for r in rs]
        return (sum(s["attn_launches"] + s["index_launches"] for s in st), sum(s["triggers"] for s in st),
                sum(s["index_launches"] for s in st))

    def timed(n, host=None, i0=0, rs=None):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        w0 = time.perf_counter()
        e0.record(sc)
        for i in range(n):
            one_step(i0 + i, host, rs)
        sc.wait_stream(sf)                                  # side-band work still in flight belongs to the region
        e1.record(sc)
        enq = time.perf_counter() - w0                      # host time to enqueue the n steps (no waiting)
        sf.synchronize(); sc.synchronize()
        w1 = time.perf_counter()
        barrier()
        ms = max_over_ranks(e0.elapsed_time(e1), dev)       # the job's time = the slowest rank's
        return ms, w1 - w0, enq, (w0, w1)

    # ---- warm-up, then the device-resident timed region ----
    clk = ClockSampler(local_rank)
    clk.start()
    for i in range(warmup):
        one_step(i)
    i_next = warmup
    l0, t0_, x0 = counters(reps)
    # a window shorter than one trigger period of every replica would hold 0 or 1 trigger, i.e. none or several times the
    # workload's share (one per tau steps and replica): at least R * tau steps are timed, whatever --steps asks for
    n_timed = max(args.steps, R * c.tau) if R * c.tau <= 8192 else args.steps
    steps_requested, args.steps = args.steps, n_timed
    ms, wall, enq, window = timed(args.steps, i0=i_next)
    clk.sample_now()
    clk.window = window
    i_next += args.steps
    # the host's own cost per step: a burst short enough never to fill the launch queue (in the long region above the host
    # is throttled by the device, so its enqueue time there only mirrors the device's)
    n_free = min(256, args.steps)
    _, _, enq_free, _ = timed(n_free, i0=i_next)
    i_next += n_free
    l1_, t1_, x1 = counters(reps)
    launches, triggers_timed, index_launches = l1_ - l0, t1_ - t0_, x1 - x0
    units_job = job_units(args.steps)
    value = units_job / (ms * 1e-3)

    # ---- end to end through the C ABI with host buffers (H2D + D2H inside the timed region) ----
    # Every step's q, k_new, v_new (and h at trigger steps) are pulled out of pinned host memory and its result lands in
    # pinned host memory, where the host waits for it.  e2e: lsa_step_host_async, up to E2E_DEPTH steps in flight, each
    # with an output buffer of its own, every ticket waited for inside the region (a serving loop with several independent
    # requests in flight); e2e_sync: lsa_step_host, the host blocks on every step.
    E2E_DEPTH = 6
    pin = lambda t: t.cpu().pin_memory()
    host = dict(q=[pin(x) for x in qs], h=[pin(x) for x in hs], kn=[pin(x) for x in kns], vn=[pin(x) for x in vns],
                out=torch.empty((c.B, c.H, c.D), dtype=tdt).pin_memory())
    outs = [torch.empty((c.B, c.H, c.D), dtype=tdt).pin_memory() for _ in range(E2E_DEPTH + 1)]
    for i in range(max(3, R)):
        one_step(i_next + i, host)
    i_next += max(3, R)
    n_e2e = max(64, args.steps // 4)
    ms_sync, _, enq_e2e, _ = timed(n_e2e, host, i0=i_next)
    i_next += n_e2e

    def timed_async(n, i0):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        tickets = []
        barrier()
        e0.record(sc)
        for i in range(n):
            r = reps[(i0 + i) % R]
            t, j = r.step, (i0 + i) % NIN
            tickets.append((r, r.ctx.step_host_async(host["q"][j], host["h"][(t // c.tau) % NIN], host["kn"][j], host["vn"][j],
                                                     outs[i % len(outs)])))
            r.step += 1
            if len(tickets) > E2E_DEPTH:
                rr, tk = tickets.pop(0)
                rr.ctx.host_wait(tk)
        for rr, tk in tickets:
            rr.ctx.host_wait(tk)
        sc.wait_stream(sf)
        e1.record(sc)
        sf.synchronize(); sc.synchronize()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), dev)

    if c.B <= 4 and args.overlap == 1 and c.dtype == "bf16" and not drift_needs_host_sync:
        timed_async(max(3, R), i_next); i_next += max(3, R)
        ms_e2e = timed_async(n_e2e, i_next); i_next += n_e2e
        e2e_mode = f"lsa_step_host_async, up to {E2E_DEPTH} steps in flight, every ticket waited for inside the region"
    else:
        ms_e2e, e2e_mode = ms_sync, "lsa_step_host (the host blocks on every step)"
    es = 4 if c.dtype == "f32" else 2
    h2d = (c.B * c.H * c.D + 2 * c.B * c.D) * es + c.B * c.Dh * es // c.tau     # h crosses only at trigger steps (1 in tau)
    d2h = c.B * c.H * c.D * es
    e2e_value = job_units(n_e2e) / (ms_e2e * 1e-3)
    e2e_sync_value = job_units(n_e2e) / (ms_sync * 1e-3)
    clocks = clk.stop()

    # ---- the other step_overlap mode, on replicas of its own (every rank runs it: there are barriers inside) ----
    dependent = None
    if not args.no_dependent and c.B <= 4 and c.dtype == "bf16":
        other = 1 - args.overlap
        reps2 = [Replica(wl, shared, sc, sf, lsa, phases[r], other) for r in range(R)]
        for i in range(warmup):
            one_step(i, None, reps2)
        n_dep = max(256, min(args.steps, 4096))
        ms_d, _, _, _ = timed(n_dep, None, warmup, reps2)
        dependent = dict(step_overlap=other, value=job_units(n_dep) / (ms_d * 1e-3), unit=unit, ms_per_step=ms_d / n_dep,
                         frac_of_hbm_peak=attn_bytes / (ms_d / n_dep * 1e-3) / 1e9 / load_peaks()["hbm_gbs"], steps=n_dep,
                         note="same loop, contexts created with the other lsa_config.step_overlap (0 = the API default: q / k_new / v_new "
                              "may be produced by the work enqueued on stream_compute just before the call)")
        for r in reps2:
            r.ctx.close()
        del reps2

    # ---- the dominant kernel alone (CUDA events around single launches on its stream: no overlap with neighbours) ----
    n_prof = min(args.steps, 512)
    for r in reps:
        r.ctx.profile_enable(n_prof // R + 8)
    for i in range(n_prof):
        one_step(i_next + i)
    i_next += n_prof
    phases_ms = {}
    for r in reps:
        for ph, v in r.ctx.profile_read().items():
            d = phases_ms.setdefault(ph, dict(ms=0.0, count=0))
            d["ms"] += v["ms"]; d["count"] += v["count"]
        r.ctx.profile_enable(0)
    attn_ms = phases_ms["attention"]["ms"] / max(phases_ms["attention"]["count"], 1)
    comb_ms = phases_ms["combine"]["ms"] / max(phases_ms["combine"]["count"], 1) if phases_ms["combine"]["count"] else 0.0
    peaks = load_peaks()
    ph_dev = phases_ms.get("attention_dev", dict(ms=0.0, count=0))
    attn_dev_ms = ph_dev["ms"] / ph_dev["count"] if ph_dev["count"] else None
    stats = reps[0].ctx.stats()
    one_launch = c.B <= 4 and args.overlap == 1 and stats["attn_impl"] == 2
    # one launch of the dominant kernel per step: its average duration over the timed region is the step time of the
    # pipelined loop (the launches of consecutive steps overlap); kernel_ms_isolated = events around single launches
    launch_ms = ms / args.steps
    achieved = attn_bytes / (launch_ms * 1e-3) / 1e9
    traffic, traffic_src = stored_traffic(c.config_id, args.overlap)
    roofline = dict(bound="hbm", achieved=achieved, peak=peaks["hbm_gbs"], unit="GB/s", frac=achieved / peaks["hbm_gbs"],
                    traffic=traffic, traffic_source=traffic_src,
                    kernel=("attn_tc_small_kernel: split-K decode attention and the merge of its partials in one launch (S7 + S8)" if one_launch
                            else "attn_tc_kernel: split-K decode attention (S7); S8 in the combine kernel that follows"),
                    algorithmic_bytes_per_launch=attn_bytes, kernel_ms=launch_ms,
                    kernel_ms_how="timed region / launches of this kernel inside it (CUDA events on stream_compute), i.e. everything a step costs is charged to it",
                    kernel_ms_isolated=attn_ms, combine_ms_isolated=comb_ms, kernel_ms_device_clock_isolated=attn_dev_ms,
                    step_ms=launch_ms, frac_of_step=achieved / peaks["hbm_gbs"],
                    peak_source=peaks["source"], frac_of_nominal_8tbs=achieved / 8000.0)

    # ---- how much of the trigger side band (S1-S5) hides behind attention (SURVEY 8(d) "fetch overlap") ----
    # exposed time per trigger = tau * (mean step time over all steps - step time between triggers); hidden fraction =
    # 1 - exposed / (side-band kernel time per trigger).  With recall_lag = 1 the new table is needed by step t + 1.
    side_band = None
    if not c.stagger and c.tau >= 8 and args.steps >= 2 * R * c.tau and all(ph in phases_ms and phases_ms[ph]["count"] for ph in ("index", "residency", "fetch")):
        # bring every replica to the same trigger phase, then time windows without a trigger or a swap
        t_al = (max(r.step for r in reps) // c.tau + 1) * c.tau + 2
        for idx, r in enumerate(reps):
            while r.step < t_al:
                one_step(idx)
        nt_ms, n_win = 0.0, 6
        for _ in range(n_win):
            sf.synchronize(); sc.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(sc)
            for _s in range(c.tau - 3):                      # phases 2 .. tau - 2 of every replica: no trigger, no swap
                for idx in range(R):
                    one_step(idx)
            e1.record(sc)
            sc.synchronize()
            nt_ms += e0.elapsed_time(e1) / (R * (c.tau - 3))
            for _s in range(3):                               # tau - 1, trigger, swap: untimed
                for idx in range(R):
                    one_step(idx)
        nt_ms /= n_win
        per = {ph: phases_ms[ph]["ms"] / phases_ms[ph]["count"] for ph in ("index", "residency", "fetch")}
        side_ms = sum(per.values())
        exposed = max(0.0, c.tau * (ms / args.steps - nt_ms))   # <= 0 within noise: nothing of the side band is exposed
        side_band = dict(step_ms_all=ms / args.steps, step_ms_between_triggers=nt_ms, exposed_ms_per_trigger=exposed,
                         side_band_ms_per_trigger=side_ms, phases_ms_per_trigger=per,
                         hidden_fraction=(1.0 - exposed / side_ms) if side_ms > 0 else None, recall_lag=c.recall_lag,
                         note="hidden_fraction = 1 - exposed / side-band kernel time; recall_lag = 1 lets only the trigger step's own attention hide it")

    # ---- chunk fetch: H2D link peak (pinned cudaMemcpyAsync) and the device-pull fetch kernel ----
    fetch = None
    if rank == 0:
        src = torch.empty(256 * 2**20, dtype=torch.uint8).pin_memory()
        dst = torch.empty(256 * 2**20, dtype=torch.uint8, device=dev)
        best = 0.0
        for _ in range(6):
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); dst.copy_(src, non_blocking=True); b_.record(); torch.cuda.synchronize()
            best = max(best, src.numel() / (a.elapsed_time(b_) * 1e-3) / 1e9)
        r = reps[0]
        r.ctx.profile_enable(64)
        nb = 0
        g = np.random.default_rng(1)
        n_ch = c.n_chunks(0)
        for it in range(8):
            sel = np.full((1, c.k), -1, dtype=np.int32)
            ke = c.k_eff(0)
            sel[0, :ke] = g.choice(n_ch, size=ke, replace=False)
            b0 = r.ctx.stats()["bytes_fetched"]
            r.ctx.fetch_chunks([0], torch.from_numpy(sel).to(dev))
            r.ctx.commit_tables()
            nb += r.ctx.stats()["bytes_fetched"] - b0
        pr = r.ctx.profile_read()
        r.ctx.profile_enable(0)
        fms = pr["fetch"]["ms"]
        fetch = dict(h2d_peak_gbs=best, fetch_gbs=(nb / (fms * 1e-3) / 1e9) if fms > 0 else None,
                     frac_of_h2d_peak=(nb / (fms * 1e-3) / 1e9 / best) if fms > 0 else None, bytes=nb, kernel_ms=fms,
                     mode="device-pull kernel over the mapped pinned cold pool",
                     residency_ms_per_trigger=pr["residency"]["ms"] / max(pr["residency"]["count"], 1))
        del src, dst

    # ---- per-CTA timeline of the small-batch launches (lsa_timeline_*; DESIGN 7.3): a stretch of its own, after the timed legs of the main
    # contexts (and before the legs that move them to other kernels: lsa_step_graph keeps a context on the general path)
    timeline = None
    if args.timeline and args.overlap and c.B <= 4 and stats["attn_impl"] == 2:
        for r in reps:
            r.ctx.timeline_enable(True)
        n_tl = 2 * R * c.tau
        for i in range(R * 8):                      # the stamps themselves are part of what is measured: settle first
            one_step(i_next + i)
        i_next += R * 8
        ms_tl, _, _, _ = timed(n_tl, i0=i_next)
        i_next += n_tl
        tl = [r.ctx.timeline_read()[0] for r in reps]
        for r in reps:
            r.ctx.timeline_enable(False)
        timeline = summarise_timeline(tl, ms_tl / n_tl)

    # ---- optional: the paper-exact Level-1 indexer (NEXT-1) at this config's context length ----
    l1 = None
    if args.l1 and rank == 0 and c.dtype == "bf16" and c.C == 128:
        from paper_2606_09079_b200.workloads import L1Inputs
        L, d_c = 3, 2048                                   # paper: layers {10,12,20}, low-rank query dim r = 2048
        l1in = L1Inputs(wl, n_layers=L, d_c=d_c)
        r = reps[0]
        layers = [{k_: to_torch(v, "bf16").to(dev) for k_, v in lay.items()} for lay in l1in.layers]
        index_k = [[to_torch(K, "bf16").to(dev) for K in l1in.index_k[b]] for b in range(c.B)]
        r.ctx.l1_init(layers, index_k, d_c=d_c)
        hd = to_torch(wl.h(0), c.dtype).to(dev)
        ids = list(range(c.B))
        for _ in range(3):
            r.ctx.l1_select(hd, ids, want_scores=False)
        r.ctx.sync()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_it = 20
        e0.record(sf)
        for _ in range(n_it):
            r.ctx.l1_select(hd, ids, want_scores=False)
        e1.record(sf)
        sf.synchronize()
        l1_ms = e0.elapsed_time(e1) / n_it
        key_bytes = sum(c.n_csa(b) for b in range(c.B)) * 128 * 2 * L
        w_bytes = L * (d_c * c.Dh + 64 * 128 * d_c + 64 * c.Dh) * 2
        l1 = dict(ms_per_trigger=l1_ms, layers=L, d_c=d_c, c_I=128, n_h=64, index_key_bytes=key_bytes, weight_bytes=w_bytes,
                  gbs=(key_bytes + w_bytes) / (l1_ms * 1e-3) / 1e9, frac_of_hbm_peak=(key_bytes + w_bytes) / (l1_ms * 1e-3) / 1e9 / load_peaks()["hbm_gbs"],
                  note="Eq.(1)-(5),(13) for all sequences of the config, warm L2 for the weights (same call repeated)")

    # ---- optional: the step with Level 2 (NEXT-2): lsa_step_l2 through the same replica rotation ----
    level2 = None
    if args.l2 and rank == 0 and c.dtype == "bf16" and c.C == 128 and stats["attn_impl"] == 2:
        from paper_2606_09079_b200.workloads import L2Inputs
        l2in = L2Inputs(wl)
        ik = [to_torch(K, "bf16").to(dev) for K in l2in.index_k]
        for r in reps:
            r.ctx.l2_init(ik, args.l2_k2)
        qis = [to_torch(l2in.q_idx(i), "bf16").to(dev) for i in range(NIN)]
        wis = [torch.from_numpy(l2in.w_idx(i)).to(dev) for i in range(NIN)]

        def l2_step(i):
            r = reps[i % R]
            t, j = r.step, i % NIN
            r.ctx.step_l2(qs[j], hs[(t // c.tau) % NIN], kns[j], vns[j], qis[j], wis[j], out)
            r.step += 1
        for i in range(max(3, 2 * R)):
            l2_step(i_next + i)
        i_next += max(3, 2 * R)
        n_l2 = max(256, args.steps // 4)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(sc)
        for i in range(n_l2):
            l2_step(i_next + i)
        e1.record(sc)
        sf.synchronize(); sc.synchronize()
        i_next += n_l2
        l2_ms = e0.elapsed_time(e1) / n_l2
        # the two Level-2 kernels alone (score + Top-k), same rotation
        e0.record(sc)
        for i in range(n_l2):
            reps[i % R].ctx.l2_select(qis[i % NIN], wis[i % NIN], want_entries=False)
        e1.record(sc)
        sc.synchronize()
        sel_ms = e0.elapsed_time(e1) / n_l2
        key_bytes = sum(c.k_eff(b) for b in range(c.B)) * c.C * 128 * 2
        level2 = dict(value=per_step_units / (l2_ms * 1e-3), unit=unit, ms_per_step=l2_ms, k2=args.l2_k2,
                      resident_entries=sum(c.k_eff(b) for b in range(c.B)) * c.C, select_ms=sel_ms, index_key_bytes_per_step=key_bytes,
                      note="lsa_step_l2: Level-2 score + Top-k2 + masked attention (S6 / append folded in) + combine; select_ms = the two Level-2 kernels alone, PDL-chained")

    # ---- optional: KV export into the cold pool (NEXT-4, first half) against the pinned D2H copy rate ----
    export = None
    if args.export and rank == 0 and not args.cold_fp8:
        n_ch = min(c.n_chunks(0), max(1, (256 * 2**20) // c.page_bytes))
        src = shared["cold"][0][:n_ch].to(dev)                   # the same bytes go back: the pool's content is unchanged
        nb = src.numel() * src.element_size()
        dstp = torch.empty(nb, dtype=torch.uint8).pin_memory()
        flat = src.view(torch.uint8).reshape(-1)
        best_d2h = 0.0
        for _ in range(5):
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); dstp.copy_(flat, non_blocking=True); b_.record(); torch.cuda.synchronize()
            best_d2h = max(best_d2h, nb / (a.elapsed_time(b_) * 1e-3) / 1e9)
        best_exp = 0.0
        for _ in range(5):
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(sf); reps[0].ctx.export_chunks(0, 0, src); b_.record(sf); sf.synchronize()
            best_exp = max(best_exp, nb / (a.elapsed_time(b_) * 1e-3) / 1e9)
        export = dict(bytes=nb, chunks=n_ch, export_gbs=best_exp, d2h_peak_gbs=best_d2h, frac_of_d2h_peak=best_exp / best_d2h,
                      mode="device kernel storing over the mapped pinned cold pool")
        del src, dstp

    # ---- optional: the step with a growing compressed history (NEXT-4, second half): lsa_append_compressed every 4th step
    # (CSA entry; HCA entry every 128th), chunks completing every 512 steps and being exported, against the static loop ----
    growth = None
    if args.growth and rank == 0 and not args.cold_fp8:
        n_gr = max(2048, min(args.steps, 8192))
        n_gr += (-n_gr) % (R * c.tau)
        per_rep = (R * c.tau * 2 + n_gr) // R + 8
        extra = per_rep // (c.csa_ratio * c.C) + 2
        cold_cap = []
        for b in range(c.B):                                # one capacity-sized cold pool per sequence, shared by the replicas
            x = torch.zeros((c.n_chunks(b) + extra,) + tuple(shared["cold"][b].shape[1:]), dtype=tdt).pin_memory()
            x[: c.n_chunks(b)] = shared["cold"][b]
            cold_cap.append(x)
        greps = []
        for ridx in range(R):
            g_ = types.SimpleNamespace()
            g_.hot_pool = torch.zeros((c.hot_pages + 2 * c.B, 2, c.C, c.D), dtype=tdt, device=dev)
            g_.emb = [torch.cat([e, torch.zeros((extra, c.E), dtype=tdt, device=dev)]) for e in shared["emb"]]
            g_.hca_k = [torch.cat([x, torch.zeros((per_rep // c.hca_ratio + 2, c.D), dtype=tdt, device=dev)]) for x in shared["hca_k"]]
            g_.hca_v = [torch.cat([x, torch.zeros((per_rep // c.hca_ratio + 2, c.D), dtype=tdt, device=dev)]) for x in shared["hca_v"]]
            g_.win_k = [x.clone() for x in shared["win_k"]]
            g_.win_v = [x.clone() for x in shared["win_v"]]
            phase = (c.tau - ridx * (c.tau // R)) % c.tau
            seqs = [dict(cold_csa=cold_cap[b], n_csa=c.n_csa(b), n_hca=c.n_hca(b), chunk_emb=g_.emb[b], hca_k=g_.hca_k[b],
                         hca_v=g_.hca_v[b], win_k=g_.win_k[b], win_v=g_.win_v[b], w_len=min(c.W, c.L[b]), w_head=0, step0=c.step0(b) + phase,
                         cap_csa=(c.n_chunks(b) + extra) * c.C, cap_hca=int(g_.hca_k[b].shape[0])) for b in range(c.B)]
            g_.ctx = lsa.LsaContext(dtype=lsa.LSA_F32 if c.dtype == "f32" else lsa.LSA_BF16, H=c.H, D=c.D, C_=c.C, W=c.W, Dh=c.Dh,
                                    E=c.E, k=c.k + 2, tau=c.tau, hot_pool=g_.hot_pool, W_q=shared["W_q"], seqs=seqs,
                                    recall_lag=c.recall_lag, stream_compute=sc, stream_fetch=sf, attn_impl=shared["attn_impl"],
                                    step_overlap=args.overlap)
            g_.step, g_.bound = phase, {}
            greps.append(g_)
        ids_all = list(range(c.B))
        emb_new = torch.nn.functional.normalize(torch.randn((c.B, c.E), device=dev, generator=torch.Generator(dev).manual_seed(c.seed)), dim=-1).to(tdt)
        n_app = [0, 0]

        def grow_step(i):
            r = greps[i % R]
            t = r.step - ((c.tau - (i % R) * (c.tau // R)) % c.tau)          # decode steps this replica has made
            j = i % NIN
            if t > 0 and t % c.csa_ratio == 0:
                hk = t % c.hca_ratio == 0
                r.ctx.append_compressed(ids_all, kns[j], vns[j], kns[j] if hk else None, vns[j] if hk else None, emb_new)
                n_app[0] += c.B; n_app[1] += c.B if hk else 0
            key = (j, (r.step // c.tau) % NIN)
            fn = r.bound.get(key)
            if fn is None:
                fn = r.bound[key] = r.ctx.bind_step(qs[j], hs[key[1]], kns[j], vns[j], out)
            fn()
            r.step += 1

        for i in range(2 * R * c.tau):
            grow_step(i)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a0 = list(n_app)
        e0.record(sc)
        for i in range(n_gr):
            grow_step(2 * R * c.tau + i)
        sc.wait_stream(sf)
        e1.record(sc)
        sf.synchronize(); sc.synchronize()
        gms = e0.elapsed_time(e1) / n_gr
        gst = [r.ctx.stats() for r in greps]
        growth = dict(value=per_step_units / (gms * 1e-3), unit=unit, ms_per_step=gms, steps=n_gr, static_ms_per_step=ms / args.steps,
                      csa_entries_in_region=n_app[0] - a0[0], hca_entries_in_region=n_app[1] - a0[1],
                      chunks_exported=sum(s_["chunks_exported"] for s_ in gst), k=c.k + 2,
                      note="k + 2 table slots and 2 B more pages, so the same k chunks are recalled as in the static loop and the tail "
                           "chunk is attended on top; an append that only writes rows runs beside the previous attention launch and the next "
                           "launch waits for its counter; a completed chunk / new tail (twice per 512 steps) is stream-ordered")
        for r in greps:
            r.ctx.close()
        del greps, cold_cap

    # ---- optional: lsa_step_graph (NEXT-3) through the same replica rotation, fixed input buffers ----
    graph = None
    if args.graph and rank == 0 and stats["attn_impl"] == 2:
        def g_step(i):
            r = reps[i % R]
            t = r.step
            r.ctx.step_graph(qs[0], hs[(t // c.tau) % NIN], kns[0], vns[0], out)
            r.step += 1
        for i in range(max(3, 2 * R)):
            g_step(i_next + i)
        i_next += max(3, 2 * R)
        n_g = max(256, args.steps // 2)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        w0 = time.perf_counter()
        e0.record(sc)
        for i in range(n_g):
            g_step(i_next + i)
        e1.record(sc)
        enq_g = time.perf_counter() - w0
        sf.synchronize(); sc.synchronize()
        i_next += n_g
        g_ms = e0.elapsed_time(e1) / n_g
        gs = [r.ctx.graph_stats() for r in reps]
        graph = dict(value=per_step_units / (g_ms * 1e-3), unit=unit, ms_per_step=g_ms, host_enqueue_ms_per_step=enq_g * 1e3 / n_g,
                     captures=sum(g_["captures"] for g_ in gs), replays=sum(g_["replays"] for g_ in gs),
                     note="lsa_step_graph: steps without a trigger or a table swap replay one captured graph (attention + combine) per context")

    cpu_baseline = cpu_baseline_1t = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n, secs, threads = oracle_sample(wl, budget_s=12.0, max_steps=24)
        cpu_baseline = dict(value=n * per_step_units / secs, unit=unit, cores=threads, kind="oracle",
                            sample=f"oracle steps 0..{n - 1} of {c.name}: trigger + fetch at step 0, attention every step; {secs:.1f} s")
        n1, secs1, _ = oracle_sample(wl, budget_s=10.0, max_steps=6, threads=1)
        cpu_baseline_1t = dict(value=n1 * per_step_units / secs1, unit=unit, cores=1, kind="oracle",
                               sample=f"oracle steps 0..{n1 - 1} of {c.name} with the BLAS pool limited to one thread; {secs1:.1f} s")

    if rank == 0:
        line = dict(metric=name, value=value, unit=unit, n_gpus=world, steps=args.steps, steps_requested=steps_requested, warmup=warmup,
                    ms_per_step=ms / args.steps, higher_is_better=True, scaling="strong" if sharded else "weak", vs_baseline=None,
                    dtype=c.dtype, data="synthetic", config=workload_config(cfg, world, l2),
                    run=dict(step_overlap=args.overlap, cold_format="fp8_e4m3" if args.cold_fp8 else "native", attn_impl={1: "simt", 2: "tcgen05"}.get(stats["attn_impl"], "?"), attn_ctas=stats["attn_ctas"],
                             replicas=R, replica_trigger_phases=phases, sequences_this_rank=c.B,
                             note="step_overlap = 1: the timed steps belong to independent layer-state replicas and their inputs are staged before the loop"),
                    e2e=dict(value=e2e_value, unit=unit, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h, steps=n_e2e,
                             ms_per_step=ms_e2e / n_e2e, mode=e2e_mode,
                             sync=dict(value=e2e_sync_value, ms_per_step=ms_sync / n_e2e, mode="lsa_step_host: the host blocks on every step")),
                    gpu_launches=int(launches), triggers_in_timed_region=int(triggers_timed), index_launches=int(index_launches),
                    tie_triggers_seen=n_tie_triggers[0], clocks=clocks, roofline=roofline, dependent_inputs=dependent,
                    cpu_baseline=cpu_baseline, cpu_baseline_1t=cpu_baseline_1t,
                    phases_ms={k_: (v["ms"] / v["count"] if v["count"] else None) for k_, v in phases_ms.items()},
                    fetch=fetch, side_band=side_band, timeline=timeline, l1_indexer=l1, level2=level2, step_graph=graph, export=export, growth=growth, wall_s=wall,
                    host_enqueue_ms_per_step=enq_free * 1e3 / n_free, host_enqueue_ms_per_step_e2e=enq_e2e * 1e3 / n_e2e,
                    tokens_per_s=(units_job if tokens else units_job * (cfg.B if sharded else c.B)) / (ms * 1e-3))
        print(json.dumps(line))
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
