#!/usr/bin/env python
"""bench.py -- EMC iterations/s of the CUDA hot path on synthetic data shaped like the paper's.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--impl ours|reference]

Default workload: BASELINE.json configs[2] = C3 (128^3 model, 128x128 detector, R = 25 000, N = 50 000), the
config BASELINE.json calls "tensor-core-bound likelihood and update" and the largest one-iteration config
that is resident on one GPU (BASELINE.json's metric names no config); C1, C2, C4, C5 by --config.
A "step" is one pass of the whole hot path over the config's workload: every EMC iteration the
config names (C3: one, C2: three, C5: five with a growing rotation list), each iteration = Expand ->
log-likelihood -> normalise -> update -> Compress, through the C ABI (emc_iterate).

Prints ONE JSON line (rank 0).  `value` = iterations/s with all inputs resident in HBM; `e2e` = the
same through the C-ABI call with HOST buffers (pinned counts streamed by the library, model and
geometry copied in, model and log-likelihood copied out inside the timed region); `roofline` is
for the dominant kernel, timed live with CUDA events recorded by the library on the launching
stream (EMC_PROFILE_STAGES); `comparator` is cuBLAS (torch.matmul, fp16) on the same operands, timed
beside it; `cpu_baseline` is the CPU oracle timed on this box's host cores on a bounded sample
(N = 1 only).  With --gpus N > 1 (torchrun) the path does not shard (north_star: one GPU, no
collectives): every rank runs an independent replica, scaling = "weak".
`--impl reference` times the oracle itself (rank 0 only): every step is one bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import pathlib
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = pathlib.Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import numpy as np  # noqa: E402

METRIC = "emc_iterations_per_s"
UNIT = "iterations/s"
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernels, from the committed `ncu --set full`
# captures (profiles/*.md name the commands); keyed "<config>:<stage>"
TRAFFIC_FILE = ROOT / "profiles" / "r02_dram_traffic.csv"       # from the committed ncu capture (profiles/r02_full_ncu.md)
TRAFFIC_COMMIT = "ca8073a"                                      # the commit that capture was taken at (emc_gemm.cu unchanged since)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=12)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C3", help="C1..C5 (BASELINE.json configs[0..4]); default C3 = configs[2]")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--weighted", action="store_true", help="Compress by eq. (2.12) instead of eq. (2.10)")
    ap.add_argument("--null-weights", action="store_true", help="pass weight = NULL (1/R) instead of the explicit equal weights")
    ap.add_argument("--gaussian-sigma", type=float, default=0.0,
                    help="> 0: time the paper's Gaussian likelihood with fluence (emc_iterate_gaussian, DESIGN.md section 11) "
                         "instead of the Poisson path; not the BASELINE.json metric, no cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true",
                    help="skip the `configs` sub-records (C1 with the step in a CUDA graph, C2, C4, C5) that the default "
                         "single-GPU C3 run adds to its line")
    ap.add_argument("--no-comparator", action="store_true", help="skip the cuBLAS fp16 GEMM on the same operands")
    ap.add_argument("--cuda-graph", action="store_true",
                    help="capture the whole step into one CUDA graph and replay it for `value` (the launch-bound C1); "
                         "per-stage times then come from a separate un-captured pass")
    ap.add_argument("--sparse", action="store_true",
                    help="side measurement: stages 2 and 4 from photon lists (EMC_SPARSE_PHOTONS) instead of the dense contractions")
    ap.add_argument("--rot-chunk", type=int, default=0,
                    help="side measurement: emc_iterate_rot_chunked with this many rotations per chunk (one pattern chunk)")
    ap.add_argument("--shard-rotations", action="store_true",
                    help="side measurement (N > 1): ONE job with the rotation list sharded over the ranks "
                         "(paper_1409_4256_b200.parallel, NCCL all-gather + all-reduce) instead of N replicas; strong scaling")
    ap.add_argument("--photons", type=float, default=0.0, help="override the config's mean photons per pixel (density sweeps)")
    ap.add_argument("--n-pat", type=int, default=0, help="override the config's pattern count (side measurements)")
    return ap.parse_args()


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return dict(hbm=d["hbm_gbs"], bf16_burst=d["bf16_tflops"], bf16_sustained=d["bf16_tflops_sustained"],
                    source="measured")
    # fallback stated by /opt/skills/guides/B200_PROFILING.md
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, source="fallback")


# ------------------------------------------------------------------------------ CPU oracle leg

def oracle_sample(inp, stage, n_rot_s, n_pat_s):
    """Times the oracle's five stages on a bounded sample and extrapolates one full iteration.  Stages 1 and 5 are linear in
    R.  Stages 2-4 are timed at TWO rotation counts (R_s and R_s / 2) on the same patterns and fitted as
    t = a N P + b R N P: oracle.loglik and oracle.update convert the whole count sample to float64 on every call, a cost that
    does not depend on R and that a purely bilinear extrapolation would multiply by R / R_s (the two arms of bench.py, which
    sample different R_s, then disagree by up to 2x).  Returns (seconds_full, dict)."""
    from oracle import emc_oracle as o

    cfg = inp.cfg
    quat, wgt = inp.quat[stage], inp.weight[stage]
    n_rot, n_pat = len(quat), cfg.n_pat
    rs, ns = min(n_rot, n_rot_s), min(n_pat, n_pat_s, inp.counts.shape[0])
    r2 = max(1, rs // 2)
    qs = quat[:rs]
    ws = (wgt[:rs] / wgt[:rs].sum()).astype(np.float32)
    ks = inp.counts[:ns]
    t = {}
    t0 = time.perf_counter()
    w, idx = o.expand(inp.model_init, inp.q, qs)
    t["expand"] = time.perf_counter() - t0

    def stages_2_to_4(rows):
        tt = {}
        t0 = time.perf_counter()
        big_l, _ = o.loglik(w[:rows], idx[:rows], ks, inp.mask)
        tt["loglik"] = time.perf_counter() - t0
        t0 = time.perf_counter()
        p, _, _ = o.normalize(big_l.astype(np.float32), (ws[:rows] / ws[:rows].sum()).astype(np.float32))
        tt["normalize"] = time.perf_counter() - t0
        t0 = time.perf_counter()
        wn, s = o.update(p.astype(np.float32), ks, inp.mask)
        tt["update"] = time.perf_counter() - t0
        return tt, wn, s

    half, _, _ = stages_2_to_4(r2)
    whole, wn, s = stages_2_to_4(rs)
    t.update(whole)
    t0 = time.perf_counter()
    o.compress(wn, inp.q, qs, inp.mask, cfg.n, slice_w=(s > 0).astype(np.float32))
    t["compress"] = time.perf_counter() - t0
    full = (t["expand"] + t["compress"]) * n_rot / rs
    fit = {}
    for k in ("loglik", "normalize", "update"):
        slope = max(0.0, (whole[k] - half[k]) / max(1, rs - r2)) if rs > r2 else whole[k] / rs     # seconds per rotation
        fixed = max(0.0, whole[k] - slope * rs)                                                   # R-independent part
        fit[k] = dict(per_rotation=slope, fixed=fixed)
        full += (fixed + slope * n_rot) * n_pat / ns
    return full, dict(times=t, times_half=half, fit=fit, sample_seconds=sum(t.values()) + sum(half.values()),
                      n_rot_sample=rs, n_pat_sample=ns)


def sample_sizes(cfg, scale=1.0):
    """Bounded sample of the workload: at most 2e7 (rotation, pixel) samples for Expand / Compress (C2's whole count)
    and 1.2e12 multiply-adds for the float64 matmuls of stages 2 and 4: 10-30 s of oracle work on 8-16 host cores
    (`scale` shrinks both for the reference arm, which repeats the sample every step)."""
    n_rot_s = int(min(max(cfg.n_rot), max(256, scale * 2.0e7 / cfg.n_pix)))
    n_pat_s = int(max(64, min(cfg.n_pat, scale * 1.2e12 / (3.0 * n_rot_s * cfg.n_pix))))
    return n_rot_s, n_pat_s


def host_threads():
    try:
        from threadpoolctl import threadpool_info

        n = [i.get("num_threads", 1) for i in threadpool_info() if i.get("user_api") == "blas"]
        return max(n) if n else 1
    except Exception:
        return 1


def cpu_baseline(inp, scale=1.0):
    cfg = inp.cfg
    n_rot_s, n_pat_s = sample_sizes(cfg, scale)
    total, parts = 0.0, []
    for stage in range(cfg.n_iter):
        if stage > 0 and cfg.n_rot[stage] == cfg.n_rot[stage - 1]:
            full = parts[-1]["full"]                        # same rotation list: same cost
        else:
            full, info = oracle_sample(inp, stage, n_rot_s, n_pat_s)
            parts.append(dict(full=full, **info))
        total += full
    value = cfg.n_iter / total
    sample = (f"oracle/emc_oracle.py stage by stage on the first {parts[0]['n_rot_sample']} rotations x "
              f"{parts[0]['n_pat_sample']} patterns x all {cfg.n_pix} pixels of {cfg.name} "
              f"({sum(p['sample_seconds'] for p in parts):.1f} s of CPU work), extrapolated linearly in R "
              f"(expand, compress) and as (a + b R) N (loglik, normalize, update; a, b fitted from the sample and its first "
              f"half of the rotations) to the full workload")
    return dict(value=value, unit=UNIT, cores=host_threads(), kind="oracle", sample=sample)


def run_reference(args):
    """The oracle as it stands on the host cores: every step times one bounded sample of the workload (steps and
    ms_per_step describe exactly that); `value` extrapolates the mean step to the full workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from emc_inputs import CONFIGS, make_inputs

    cfg = CONFIGS[args.config]
    scale = 0.3
    _, n_pat_s = sample_sizes(cfg, scale)
    inp = make_inputs(cfg, n_pat=min(cfg.n_pat, max(n_pat_s, 512)))
    inp.cfg = cfg                                           # extrapolate to the full pattern count
    warm = max(args.warmup, 1)
    times, values = [], []
    base = None
    for i in range(warm + args.steps):
        t0 = time.perf_counter()
        base = cpu_baseline(inp, scale)
        if i >= warm:
            times.append(time.perf_counter() - t0)
            values.append(base["value"])
    value = statistics.mean(values)
    base = dict(base, value=value)
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=warm, ms_per_step=1e3 * statistics.mean(times), higher_is_better=True,
                scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=bench_config(cfg, int(os.environ.get("WORLD_SIZE", "1")), args.weighted, args.null_weights,
                                    int(np.count_nonzero(inp.mask))),
                note="every step times the CPU oracle on one bounded sample (cpu_baseline.sample); ms_per_step is the wall "
                     "time of such a step, value the extrapolation to the full workload (eq. (2.10), explicit weights: the "
                     "oracle has one code path)",
                ms_per_full_step_extrapolated=1e3 * cfg.n_iter / value,
                cpu_baseline=base,
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))


def bench_config(cfg, world, weighted, null_weights, p_eff):
    """`config` of the JSON line: the same keys and values in both arms (--impl reference times the oracle on this workload)."""
    return dict(workload=workload_name(cfg), parallelism="replicas only" if world > 1 else "1 GPU",
                l2="per-iteration working set exceeds the 126 MB L2, no flush" if cfg.name != "C1"
                else "working set fits L2 (launch-latency-bound config), no flush",
                compress="eq. (2.12)" if weighted else "eq. (2.10)", p_eff=p_eff,
                weights="NULL (1/R): uniform branches, normalize_kernel<true>" if null_weights
                else "explicit equal weights: general branches, normalize_kernel<false>")


def workload_name(cfg):
    r = "->".join(str(x) for x in cfg.n_rot) if len(set(cfg.n_rot)) > 1 else str(cfg.n_rot[0])
    return (f"{cfg.name}: model {cfg.n}^3 fp32, detector {cfg.n_det}x{cfg.n_det}, R={r}, N={cfg.n_pat} "
            f"{cfg.count_dtype} patterns at {cfg.mean_photons} photons/pixel, {cfg.n_iter} iteration(s)"
            + (f", pattern chunks of {cfg.n_pat_chunk}" if cfg.n_pat_chunk < cfg.n_pat else ""))


# ------------------------------------------------------------------------------ clocks

class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index):
        import torch

        self.path = tempfile.NamedTemporaryFile(prefix="emc_clocks_", suffix=".csv", delete=False).name
        sel = str(device_index)
        try:
            sel = "GPU-" + str(torch.cuda.get_device_properties(device_index).uuid)
        except Exception:
            pass
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", sel, f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
            time.sleep(0.3)                                 # let the sampler start before the timed region does
        except Exception:
            pass

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in open(self.path).read().splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        os.unlink(self.path)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        # "under load": the samples in the upper half of the power range (the sampler also sees the idle edges)
        lo, hi = min(power), max(power)
        load = [c for c, w in zip(sm, power) if w >= lo + 0.5 * (hi - lo)] or sm
        return dict(sm_mhz=statistics.median(load), sm_max_mhz=max(smax), power_w_max=max(power), samples=len(sm),
                    reasons=sorted(reasons))


# ------------------------------------------------------------------------------ replicas

def whole_job(ms_local, units_per_rank, world, device):
    """The path does not shard: every rank runs a replica.  Returns (max over ranks of the device
    time in ms, whole-job rate = units all ranks processed / that time).  The only collective of a run."""
    ms = float(ms_local)
    if world > 1:
        import torch
        import torch.distributed as dist

        t = torch.tensor([ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return ms, world * units_per_rank / (ms * 1e-3)


# ------------------------------------------------------------------------------ cuBLAS on the same operands

def cublas_comparator(emc, torch, d_model0, d_q, d_mask, quat, d_counts, n_rep=4):
    """The log-likelihood contraction's operands handed to cuBLAS: hi plane of log W (fp16, [R, P], masked pixels 0)
    times the count matrix (fp16, [N, P]) -> [R, N], torch.matmul, CUDA events.  ONE plane: the kernel issues two
    such products per launch, so its ISSUED rate is what compares with this number.  The count operand is mostly
    zeros, which lowers the tensor cores' switching power; a dense random GEMM (MEASURED_PEAKS.json) does not have
    that advantage, this one does."""
    w, _ = emc.emc_expand(d_model0, d_q, quat, want_idx=False)
    a = torch.log(torch.clamp(w, min=1e-30))
    del w
    a *= d_mask.to(torch.float32)[None, :]
    a = a.to(torch.float16)
    b = torch.empty(d_counts.shape, dtype=torch.float16, device="cuda")
    for d0 in range(0, d_counts.shape[0], 8192):           # in slices: no int32 copy of the whole matrix
        b[d0:d0 + 8192] = (d_counts[d0:d0 + 8192].to(torch.int32) * d_mask.to(torch.int32)[None, :]).to(torch.float16)
    torch.cuda.synchronize()
    c = None
    for _ in range(2):
        c = torch.matmul(a, b.t())
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n_rep):
        c = torch.matmul(a, b.t())
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / n_rep
    flops = 2.0 * a.shape[0] * b.shape[0] * a.shape[1]
    del a, b, c
    torch.cuda.empty_cache()
    return dict(what="torch.matmul (cuBLAS) fp16 [R,P] x [N,P]^T on the hi plane of log W and the count matrix of this "
                     "workload, all P pixels, fp16 output", ms=ms, tflops=flops / (ms * 1e-3) / 1e12, reps=n_rep)


# ------------------------------------------------------------------------------ our arm

def other_configs(args):
    """Sub-records of the other BASELINE.json configs for the default line: each is this same script run on that config in
    a process of its own (before the headline measurement allocates anything), so the numbers of DESIGN.md section 9's
    table come from the same driver-timed run as `value`.  A config that fails or runs out of time is recorded as such."""
    import subprocess

    subs = {}
    for name, extra, steps in (("C1", ["--cuda-graph"], 50), ("C2", [], 20), ("C4", [], 3), ("C5", [], 3)):
        cmd = [sys.executable, str(ROOT / "bench.py"), "--config", name, "--steps", str(steps), "--warmup", "3",
               "--no-cpu-baseline", "--no-comparator", "--no-configs"] + extra
        t0 = time.perf_counter()
        try:
            r = subprocess.run(cmd, capture_output=True, text=True, timeout=240)
            d = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1])
            subs[name] = dict(workload=d["config"]["workload"], value=d["value"], unit=d["unit"], steps=d["steps"],
                              ms_per_step=d["ms_per_step"], e2e=d["e2e"]["value"], gpu_launches=d["gpu_launches"],
                              stage_ms={k: v["ms"] for k, v in d["stages"].items()}, clocks=d["clocks"],
                              loglik_per_iteration=d["loglik_per_iteration"], cuda_graph=bool(extra),
                              roofline_frac=d["roofline"]["frac"], wall_s=time.perf_counter() - t0)
        except Exception as e:                                      # noqa: BLE001  (reported, never fatal for the headline)
            subs[name] = dict(error=f"{type(e).__name__}: {str(e)[:200]}", wall_s=time.perf_counter() - t0)
    return subs


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    configs_extra = None
    if (args.config == "C3" and not args.no_configs and int(os.environ.get("WORLD_SIZE", "1")) == 1 and args.gpus == 1
            and not (args.sparse or args.rot_chunk or args.cuda_graph or args.gaussian_sigma > 0 or args.photons > 0 or args.n_pat > 0)):
        configs_extra = other_configs(args)

    from emc_inputs import CONFIGS, make_inputs

    import dataclasses

    cfg = CONFIGS[args.config]
    if args.photons > 0:
        cfg = dataclasses.replace(cfg, mean_photons=args.photons)
    if args.n_pat > 0:
        cfg = dataclasses.replace(cfg, n_pat=args.n_pat, n_pat_chunk=min(cfg.n_pat_chunk, args.n_pat))
    inp = make_inputs(cfg)                                   # every rank: an independent replica

    import torch
    import torch.distributed as dist

    import paper_1409_4256_b200 as emc

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = measured_peaks()
    warmup = max(args.warmup, 3)

    dev = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    q2d = inp.q.reshape(cfg.n_det, cfg.n_det, 3)           # row-major 2-D detector: emc_detector.row_len = n_det
    d_model0, d_q, d_mask, d_counts = dev(inp.model_init), dev(q2d), dev(inp.mask), dev(inp.counts)
    # consecutive iterations on the same rotation list go into one emc_iterate call
    plan = []
    for s in range(cfg.n_iter):
        if plan and cfg.n_rot[s] == cfg.n_rot[s - 1]:
            plan[-1][2] += 1
        else:
            plan.append([dev(inp.quat[s]), None if args.null_weights else dev(inp.weight[s]), 1, inp.quat[s], inp.weight[s]])
    flags = emc.EMC_COMPRESS_WEIGHTED if args.weighted else 0
    if args.sparse:
        flags |= emc.EMC_SPARSE_PHOTONS
    chunk = cfg.n_pat_chunk if cfg.n_pat_chunk < cfg.n_pat else 0
    ws_bytes = max(emc.emc_workspace_bytes(cfg.n, cfg.n_pix, r, cfg.n_pat_chunk, emc.EMC_PATTERNS_ON_HOST | flags)
                   for r in cfg.n_rot)
    if args.rot_chunk > 0:
        ws_bytes = max(ws_bytes, max(emc.load().emc_workspace_bytes_rot_chunked(cfg.n, cfg.n_pix, r, args.rot_chunk, cfg.n_pat)
                                     for r in cfg.n_rot))
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda")
    ctx = emc.EmcContext()                                   # copy stream + timing events, created outside the hot path
    d_ll = torch.zeros(cfg.n_iter, dtype=torch.float64, device="cuda")
    bufs = [torch.empty_like(d_model0), torch.empty_like(d_model0)]

    def step(f):
        """all iterations of the config, device-resident inputs"""
        src, k, it0 = d_model0, 0, 0
        for quat, wgt, n_it, _, _ in plan:
            if args.gaussian_sigma > 0:
                out = emc.emc_iterate_gaussian(src, d_q, d_mask, quat, wgt, d_counts, args.gaussian_sigma, n_iter=n_it,
                                               flags=f | emc.EMC_COMPRESS_WEIGHTED, ws=ws, ctx=ctx)
                d_ll[it0:it0 + n_it] = out["loglik"]
                src, it0 = out["model"], it0 + n_it
                continue
            if args.shard_rotations and world > 1:
                from paper_1409_4256_b200 import parallel

                out = parallel.iterate_sharded(src, d_q, d_mask, quat, wgt, d_counts, n_iter=n_it, flags=f & ~emc.EMC_PROFILE_STAGES)
                d_ll[it0:it0 + n_it] = out["loglik"]
                src, it0 = out["model"], it0 + n_it
                continue
            if args.rot_chunk > 0:
                out = emc.emc_iterate_rot_chunked(src, d_q, d_mask, quat, wgt, d_counts, args.rot_chunk, n_iter=n_it, flags=f,
                                                  ws=ws, ctx=ctx)
                d_ll[it0:it0 + n_it] = out["loglik"]
                src, it0 = out["model"], it0 + n_it
                continue
            emc.emc_iterate(src, d_q, d_mask, quat, wgt, d_counts, n_iter=n_it, n_pat_chunk=chunk, flags=f, ws=ws,
                            model_out=bufs[k], loglik=d_ll[it0:it0 + n_it], ctx=ctx)
            src, k, it0 = bufs[k], 1 - k, it0 + n_it
        return src

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step(flags)
    emc.emc_check(ws)
    emc.emc_profile_read(ctx)

    clocks = ClockSampler(local)
    launches0 = emc.emc_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if args.cuda_graph:
        # the library creates nothing and never synchronises inside emc_iterate: the step is capturable as it is
        torch.cuda.synchronize()        # the workspace moves to another stream: the warm-up steps are over first
        side = torch.cuda.Stream()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            step(flags)
            launches_per_step = emc.emc_launch_count()
            with torch.cuda.graph(graph, stream=side):
                step(flags)
            launches_per_step = emc.emc_launch_count() - launches_per_step
        torch.cuda.synchronize()
        for _ in range(warmup):
            graph.replay()
        barrier()
        ev0.record()
        for _ in range(args.steps):
            graph.replay()
        ev1.record()
        barrier()
        ms = ev0.elapsed_time(ev1)
        launches = launches_per_step * args.steps
        for _ in range(args.steps):                       # per-stage times: an eager pass, not part of `value`
            step(flags | emc.EMC_PROFILE_STAGES)
        torch.cuda.synchronize()
    else:
        barrier()
        ev0.record()
        for _ in range(args.steps):
            step(flags | emc.EMC_PROFILE_STAGES)
        ev1.record()
        barrier()
        ms = ev0.elapsed_time(ev1)
        launches = emc.emc_launch_count() - launches0
    clk = clocks.stop()
    prof = emc.emc_profile_read(ctx)
    ms, value = whole_job(ms, args.steps * cfg.n_iter, world, "cuda")

    sharded = args.shard_rotations and world > 1
    if sharded:
        value /= world                       # one job, not N replicas: iterations of THE job per second
    if args.gaussian_sigma > 0 or args.sparse or args.rot_chunk > 0 or sharded:
        # a side measurement: device-resident only, per-stage CUDA-event times, no roofline / e2e / cpu legs
        prof_g = {k: v[0] / (args.steps * cfg.n_iter) for k, v in prof.items()}
        name = ("emc_gaussian_iterations_per_s" if args.gaussian_sigma > 0 else
                "emc_iterations_per_s[photon lists]" if args.sparse else
                f"emc_iterations_per_s[rotations sharded over {world} ranks, strong scaling]" if sharded else
                f"emc_iterations_per_s[rotation chunks of {args.rot_chunk}]")
        if rank == 0:
            print(json.dumps(dict(metric=name, value=value, unit=UNIT, n_gpus=world,
                                  steps=args.steps, warmup=warmup, ms_per_step=ms / args.steps,
                                  sigma=args.gaussian_sigma, config=dict(workload=workload_name(cfg)), clocks=clk,
                                  stage_ms_per_iteration=prof_g, gpu_launches=int(launches),
                                  loglik_per_iteration=[float(x) for x in d_ll.cpu().tolist()])))
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- end to end through the C ABI with HOST buffers
    h_counts = torch.from_numpy(inp.counts).pin_memory()
    h_model = torch.from_numpy(inp.model_init).pin_memory()
    h_q, h_mask = torch.from_numpy(q2d).pin_memory(), torch.from_numpy(inp.mask).pin_memory()
    h_rot = [(torch.from_numpy(np.ascontiguousarray(q)).pin_memory(), torch.from_numpy(w).pin_memory())
             for _, _, _, q, w in plan]
    h_out = torch.empty_like(h_model).pin_memory()
    h_ll = torch.empty(cfg.n_iter, dtype=torch.float64).pin_memory()
    e_model, e_q, e_mask = torch.empty_like(d_model0), torch.empty_like(d_q), torch.empty_like(d_mask)
    e_rot = [(torch.empty_like(q), torch.empty(len(w), dtype=torch.float32, device="cuda")) for q, _, _, _, w in plan]
    h2d = (h_counts.numel() * h_counts.element_size() * (cfg.n_iter if chunk else len(plan))
           + h_model.numel() * 4 + h_q.numel() * 4 + h_mask.numel()
           + sum(q.numel() * 4 + w.numel() * 4 for q, w in h_rot))
    d2h = h_out.numel() * 4 + h_ll.numel() * 8

    def step_e2e():
        e_model.copy_(h_model, non_blocking=True)
        e_q.copy_(h_q, non_blocking=True)
        e_mask.copy_(h_mask, non_blocking=True)
        src, k, it0 = e_model, 0, 0
        for (hq, hw), (dq, dw), (_, _, n_it, _, _) in zip(h_rot, e_rot, plan):
            dq.copy_(hq, non_blocking=True)
            dw.copy_(hw, non_blocking=True)
            emc.emc_iterate(src, e_q, e_mask, dq, dw, h_counts, n_iter=n_it, n_pat_chunk=chunk,
                            flags=flags | emc.EMC_PATTERNS_ON_HOST, ws=ws, model_out=bufs[k],
                            loglik=d_ll[it0:it0 + n_it], ctx=ctx)
            src, k, it0 = bufs[k], 1 - k, it0 + n_it
        h_out.copy_(src, non_blocking=True)
        h_ll.copy_(d_ll, non_blocking=True)
        torch.cuda.current_stream().synchronize()           # the user reads the result

    for _ in range(2):
        step_e2e()
    barrier()
    ev0.record()
    for _ in range(args.steps):
        step_e2e()
    ev1.record()
    barrier()
    ms_e2e = ev0.elapsed_time(ev1)
    ms_e2e, e2e_value = whole_job(ms_e2e, args.steps * cfg.n_iter, world, "cuda")

    # ---- rooflines from the live per-stage CUDA-event times
    p_eff = int(inp.mask.sum())
    rn = sum(r * cfg.n_pat for r in cfg.n_rot) * args.steps            # (rotation, pattern) pairs processed
    rp = sum(cfg.n_rot) * args.steps
    g = cfg.n ** 3
    stage_ms = {k: v[0] for k, v in prof.items()}
    stage_spans = {k: v[1] for k, v in prof.items()}
    useful = 2.0 * rn * p_eff                                           # flops of ONE contraction, all launches
    tf = lambda fl, ms_: fl / (ms_ * 1e-3) / 1e12 if ms_ > 0 else 0.0
    gbs = lambda by, ms_: by / (ms_ * 1e-3) / 1e9 if ms_ > 0 else 0.0
    stages = {
        "loglik": dict(ms=stage_ms["loglik"], launches=stage_spans["loglik"], bound="tensor",
                       useful_tflops=tf(useful, stage_ms["loglik"]),
                       issued_tflops=tf(2 * useful, stage_ms["loglik"]), planes=2, dtype="fp16x2"),
        "update": dict(ms=stage_ms["update"], launches=stage_spans["update"], bound="tensor",
                       useful_tflops=tf(useful, stage_ms["update"]),
                       issued_tflops=tf(2 * useful, stage_ms["update"]), planes=2, dtype="fp16x2 chunk-scaled"),
        "expand": dict(ms=stage_ms["expand"], bound="hbm",
                       gbs=gbs(rp * cfg.n_pix * 4.0 + 4.0 * g * stage_spans["expand"], stage_ms["expand"])),
        "normalize": dict(ms=stage_ms["normalize"], bound="hbm", gbs=gbs(8.0 * rn, stage_ms["normalize"])),
        "compress": dict(ms=stage_ms["compress"], bound="hbm",
                         gbs=gbs(rp * cfg.n_pix * 4.0 + 8.0 * g * stage_spans["compress"], stage_ms["compress"])),
        "pack": dict(ms=stage_ms["pack"]),
    }
    for k in ("expand", "normalize", "compress"):
        stages[k]["frac_of_hbm"] = stages[k]["gbs"] / peaks["hbm"]
    # which measured cuBLAS figure: the sustained one when the kernel is timed inside a long step (a timed region of a
    # second or more, where the 1 kW power cap decides the clock), the burst one for a short region
    sustained = ms >= 1000.0
    peak = peaks["bf16_sustained"] if sustained else peaks["bf16_burst"]
    for k in ("loglik", "update"):
        stages[k]["useful_frac_of_peak"] = stages[k]["useful_tflops"] / peak
        stages[k]["issued_frac_of_peak"] = stages[k]["issued_tflops"] / peak
    dom = "update" if stage_ms["update"] >= stage_ms["loglik"] else "loglik"
    traffic, traffic_src = None, None
    if TRAFFIC_FILE.exists():
        for ln in TRAFFIC_FILE.read_text().splitlines()[1:]:
            c_, s_, b_ = ln.split(",")
            if c_ == cfg.name and s_ == dom:
                traffic, traffic_src = float(b_), ("NOT measured in this run: read from the committed capture profiles/r02_full_ncu.md "
                                                   f"of commit {TRAFFIC_COMMIT} (ncu --set full, dram read + write bytes per launch)")
    # tensor-core peak the chip has at the clock it held during this run (148 SMs x 8192 dense fp16 flops per clock)
    clock_peak = 148 * 8192 * clk["sm_mhz"] * 1e6 / 1e12 if clk.get("sm_mhz") else None
    roofline = dict(bound="tensor", kernel=f"plane_gemm_pair_kernel ({dom}, {stages[dom]['dtype']})",
                    achieved=stages[dom]["useful_tflops"], peak=peak, unit="TFLOP/s",
                    frac=stages[dom]["useful_tflops"] / peak, traffic=traffic,
                    issued=stages[dom]["issued_tflops"], issued_frac=stages[dom]["issued_tflops"] / peak,
                    issued_frac_of_clock_peak=(stages[dom]["issued_tflops"] / clock_peak) if clock_peak else None,
                    clock_peak_tflops=clock_peak,
                    peak_source=f"{peaks['source']} cuBLAS bf16 " + ("sustained (timed region of %.2f s)" % (ms * 1e-3)
                                                                      if sustained else "burst (timed region of %.0f ms)" % ms),
                    avg_launch_ms=stage_ms[dom] / max(1, stage_spans[dom]),
                    traffic_unit="DRAM bytes per launch (ncu)", traffic_source=traffic_src,
                    note="achieved = ALGORITHMIC flops 2*R*N*P_eff per launch / CUDA-event launch time.  The fp16x2 split "
                         "scheme issues two tensor-core products per algorithmic one (DESIGN.md section 6): `issued` is "
                         "that MMA rate, to be read against `comparator` (cuBLAS fp16 on the same, mostly-zero count "
                         "operand) and against clock_peak_tflops = 148 SMs x 8192 flop/clk x the SM clock of this run")

    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=warmup,
                ms_per_step=ms / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="fp16x2 operand planes, f32 accumulate", data="synthetic",
                config=bench_config(cfg, world, args.weighted, args.null_weights, p_eff),
                clocks=clk,
                e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
                         ms_per_step=ms_e2e / args.steps),
                gpu_launches=int(launches),
                useful_tflops_loglik_plus_update=tf(2 * useful, stage_ms["loglik"] + stage_ms["update"]),
                roofline=roofline, stages=stages,
                loglik_per_iteration=[float(x) for x in d_ll.cpu().tolist()])
    if rank == 0:
        if world == 1 and not args.no_comparator:
            del h_counts
            line["comparator"] = cublas_comparator(emc, torch, d_model0, d_q, d_mask, plan[-1][0], d_counts)
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(inp)
        if configs_extra is not None:
            line["configs"] = configs_extra
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
