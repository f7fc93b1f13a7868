#!/usr/bin/env python
"""bench.py - one JSON line for the LTV-scan hot path (rollout + Phi/tube + adjoint) on N B200s.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]
  python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path over one batch of the workload (default: BASELINE.json
configs[1], rope N=50: n=300, m=6, T=32, batch 64 per GPU; seeded synthetic mass-spring Jacobians, see
DESIGN.md).  `value` = Phi blocks per second over the whole step, inputs resident in HBM, CUDA-event timed,
max over ranks; `e2e` = the same through ltv_scan_pipeline_host with pinned HOST buffers (H2D of every input
and D2H of x, r, lambda, grad_u, grad_x0 inside the timed region; Phi stays device-resident).
`--impl reference` times the fp64 CPU oracle on a bounded sample (rank 0 only)."""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "LTV scan rollouts/s + SLS Phi blocks/s; % of B200 tensor/HBM roofline"
UNIT = "Phi blocks/s (whole step: rollout + Phi/tube + adjoint)"
UNIT_C5 = "rollout+adjoint pairs/s"
NOMINAL_TF32_OVER_BF16 = 0.5          # dense tensor peaks, B200_PROFILING.md: tf32 1.1 vs bf16 2.25 PFLOP/s
FALLBACK_BF16_TFLOPS = 1590.0         # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent
FALLBACK_BF16_SUSTAINED = 1400.0


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="index into BASELINE.json configs (0..4)")
    ap.add_argument("--batch", type=int, default=0, help="items per GPU (0 = the config's own; config 4 sweeps 64/256/1024)")
    ap.add_argument("--quick", action="store_true",
                    help="only the headline workload: no sustained / dense legs, no other configs, no NEXT rows")
    ap.add_argument("--sustained", action="store_true", help="add the >= 2 s sustained leg (always on in the default run)")
    ap.add_argument("--next-rows", action="store_true",
                    help="add the SURVEY 8(f) calls timed alone (observer, Kalman, constraints, output feedback; p = 6)")
    ap.add_argument("--no-tf32-peak", action="store_true",
                    help="skip the live TF32 library-GEMM peak measurement (the committed figure is used instead)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-items", type=int, default=0, help="items in the CPU-oracle sample (0 = auto)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--tf32-peak", action="store_true",
                    help="only measure the TF32 library-GEMM peak (the roofline denominator) and print it")
    return ap.parse_args()


TRAFFIC_FILE = "profiles/r2_traffic.csv"


def ncu_traffic(cfg_index, kernel):
    """(dram bytes per step of `kernel`, where the figure comes from).  NOT measured in this run: ncu cannot be attached
    to a timed run, so the figure is read from the committed `ncu --set full` capture of the same kernel and workload
    (dram__bytes_read.sum + dram__bytes_write.sum summed over the launches of one step); (None, None) if that capture
    has no row for this config."""
    path = os.path.join(ROOT, TRAFFIC_FILE)
    try:
        for ln in open(path).read().splitlines()[1:]:
            c, k, b = ln.split(",")[:3]
            if int(c) == cfg_index and k == kernel:
                return float(b), f"{TRAFFIC_FILE} (committed ncu --set full capture, not measured in this run)"
    except Exception:
        pass
    return None, None


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(source="measured", hbm_gbs=p["hbm_gbs"], bf16=p["bf16_tflops"],
                    bf16_sustained=p.get("bf16_tflops_sustained", p["bf16_tflops"]))
    return dict(source="fallback", hbm_gbs=6650.0, bf16=FALLBACK_BF16_TFLOPS, bf16_sustained=FALLBACK_BF16_SUSTAINED)


class ClockSampler(threading.Thread):
    """Samples SM clock, power and throttle reasons with NVML in a tight loop (one query costs ~0.1-1 ms) and keeps
    a wall-clock stamp with every sample, so that `result(window=(t0, t1))` reports the samples that fall inside
    one timed region.  Started once, before the warm-up, so that short regions still hold several samples."""

    def __init__(self, index, period=0.002):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.stop_flag, self.max_mhz = index, period, [], False, None
        self.error = None
        self.ready = threading.Event()

    def run(self):
        try:
            import pynvml as N

            N.nvmlInit()
            h = N.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = N.nvmlDeviceGetMaxClockInfo(h, N.NVML_CLOCK_SM)
            self.names = {
                N.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                N.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                N.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                N.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            }
            self.ready.set()
            while not self.stop_flag:
                mhz = N.nvmlDeviceGetClockInfo(h, N.NVML_CLOCK_SM)
                r = N.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                try:
                    watts = N.nvmlDeviceGetPowerUsage(h) / 1e3
                except Exception:
                    watts = None
                self.samples.append((time.time(), mhz, r, watts))
                time.sleep(self.period)
        except Exception as e:  # NVML missing: report that, never fail the bench
            self.error = f"nvml_unavailable:{type(e).__name__}"
            self.ready.set()

    def result(self, window=None):
        """Median SM clock / reasons over the samples stamped inside `window` = (t0, t1) wall-clock seconds (all
        samples if None).  A window shorter than the sampling period takes the nearest sample on either side."""
        smp = list(self.samples)
        if window is not None and smp:
            t0, t1 = window
            inside = [s for s in smp if t0 <= s[0] <= t1]
            if len(inside) < 2:
                mid = 0.5 * (t0 + t1)
                inside = sorted(smp, key=lambda s: abs(s[0] - mid))[:2]
            smp = inside
        reasons = set()
        for s in smp:
            for bit, nm in getattr(self, "names", {}).items():
                if s[2] & bit:
                    reasons.add(nm)
        if self.error:
            reasons.add(self.error)
        mhz = sorted(s[1] for s in smp)
        watts = [s[3] for s in smp if s[3] is not None]
        return dict(sm_mhz=(mhz[len(mhz) // 2] if mhz else None), sm_max_mhz=self.max_mhz, reasons=sorted(reasons),
                    samples=len(mhz), power_w_max=(max(watts) if watts else None))


def measure_tf32_peak(dev, index, sustained_s=4.0, size=8192):
    """The roofline denominator of the tensor-bound kernel, measured the way MEASURED_PEAKS.json measures bf16
    (BASELINE.md section 2): torch.matmul on fp32 size^3 with TF32 allowed (a cuBLAS library
    GEMM - used ONLY as the yardstick, never on the path), 2 size^3 flop; best of 10 = burst, back to back for
    `sustained_s` seconds = sustained; SM clock / throttle reasons sampled meanwhile."""
    import torch

    old = torch.backends.cuda.matmul.allow_tf32
    torch.backends.cuda.matmul.allow_tf32 = True
    try:
        a = torch.randn((size, size), device=dev)
        b = torch.randn((size, size), device=dev)
        c = torch.empty((size, size), device=dev)
        flop = 2.0 * size ** 3
        for _ in range(3):
            torch.matmul(a, b, out=c)
        torch.cuda.synchronize()
        best = 1e30
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            torch.matmul(a, b, out=c)
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        reps = max(10, int(sustained_s / (best * 1e-3)))
        sampler = ClockSampler(index)
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        t0 = time.time()
        e0.record()
        for _ in range(reps):
            torch.matmul(a, b, out=c)
        e1.record()
        torch.cuda.synchronize()
        t1 = time.time()
        sampler.stop_flag = True
        sampler.join(timeout=2)
        sus_ms = e0.elapsed_time(e1) / reps
        del a, b, c
        return dict(tf32_tflops=flop / (best * 1e-3) / 1e12, tf32_tflops_sustained=flop / (sus_ms * 1e-3) / 1e12,
                    how=f"torch.matmul fp32 {size}^3, allow_tf32 (cuBLAS), 2 N^3 flop: best of 10 (burst); "
                        f"{reps} back to back over {t1 - t0:.1f} s (sustained)",
                    clocks_sustained=sampler.result(window=(t0, t1)))
    finally:
        torch.backends.cuda.matmul.allow_tf32 = old


def workload(cfg_index, rank, world, batch_override=None):
    """Per-rank inputs.  Weak scaling: the global batch is `batch * world` items of the same seeded workload and
    rank r owns the contiguous shard `shard_range(global, r, world)` (no data-path collective: items are
    independent); at world = 1 this is exactly BASELINE.json's config."""
    from paper_2606_14188_b200.sharding import shard_range
    from workloads import config, generate

    base = config(cfg_index)
    per_gpu = batch_override or base["batch"]
    cfg = config(cfg_index, batch=per_gpu * world)
    b0, b1 = shard_range(cfg["batch"], rank, world)
    W = generate(cfg, item_range=(b0, b1))
    cfg["batch"] = per_gpu
    return cfg, W


def cpu_oracle_step(W, items, phi_on=True):
    """One pass of the whole path by the fp64 oracle over `items` batch items; returns seconds."""
    from oracle import ltv_oracle as O

    t0 = time.perf_counter()
    for b in range(items):
        O.rollout_item(W.A[b], W.B[b], W.c[b], W.x0[b], W.u[b])
        if phi_on:
            O.system_response_tube_item(W.A[b], W.w[b])
        O.adjoint_item(W.A[b], W.B[b], W.g[b])
    return time.perf_counter() - t0


def blas_threads():
    try:
        from threadpoolctl import threadpool_info

        return max([p.get("num_threads", 1) for p in threadpool_info()] or [os.cpu_count() or 1])
    except Exception:
        return os.cpu_count() or 1


def run_reference(args, rank, world):
    if rank != 0:
        return
    cfg, W = workload(args.config, 0, 1, batch_override=max(1, args.cpu_items or (8 if args.config in (1, 2) else
                                                                                  2 if args.config == 3 else 32)))
    items = W.A.shape[0]
    from workloads import config as _config
    config_batch = _config(args.config)["batch"]
    T, n = cfg["T"], cfg["n"]
    P = T * (T - 1) // 2
    phi_on = args.config != 4
    unit = UNIT if phi_on else UNIT_C5
    for _ in range(min(args.warmup, 1)):
        cpu_oracle_step(W, 1, phi_on)
    times = [cpu_oracle_step(W, items, phi_on) for _ in range(args.steps)]
    sec = sum(times) / len(times)
    val = items * (P if phi_on else 1) / sec
    cores = blas_threads()
    line = dict(metric=METRIC, value=val, unit=unit, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=sec * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", impl="reference",
                config=dict(workload=f"{cfg['name']}: n={n} m={cfg['m']} T={T}, {items}-item sample per step "
                                     f"(full batch {config_batch})", l2="n/a (CPU)"),
                cpu_baseline=dict(value=val, unit=unit, cores=cores, kind="oracle",
                                  sample=f"{items} items of {cfg['name']} per step, whole path in fp64 numpy"),
                e2e=dict(value=val, unit=unit, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line), flush=True)


def _log(msg):
    """Progress on stderr (the JSON line on stdout stays alone)."""
    print(f"[bench {time.strftime('%H:%M:%S')}] {msg}", file=sys.stderr, flush=True)


def _events(torch):
    return torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)


class Bench:
    """Shared state of one bench.py process: device, distributed world, NVML sampler, measured peaks."""

    def __init__(self, args, rank, world, local):
        import torch
        import torch.distributed as dist

        self.args, self.rank, self.world, self.local = args, rank, world, local
        self.torch, self.dist = torch, dist
        self.dev = torch.device("cuda", local)
        self.sampler = ClockSampler(local)
        self.sampler.start()                      # before any warm-up: short regions still get several samples
        self.sampler.ready.wait(timeout=10)
        self.pk = peaks()
        self.tf32 = None

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def max_over_ranks(self, v):
        if self.world > 1:
            t = self.torch.tensor([v], device=self.dev, dtype=self.torch.float64)
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
            return float(t.item())
        return float(v)

    def tensor_peak(self, region_s):
        """(peak TFLOP/s, source): the MEASURED TF32 library-GEMM peak of this run - the burst figure for a timed region
        under one second, the sustained one otherwise; without a live measurement, the committed one of
        profiles/tf32_peak.md."""
        t = self.tf32 or dict(tf32_tflops=746.0, tf32_tflops_sustained=606.8, committed=True)
        which = "burst" if region_s < 1.0 else "sustained"
        val = t["tf32_tflops"] if which == "burst" else t["tf32_tflops_sustained"]
        src = ("profiles/tf32_peak.md (committed measurement)" if t.get("committed") else
               "measured in this run (torch.matmul fp32 8192^3, allow_tf32)")
        return val, f"TF32 library GEMM, {which} figure ({region_s:.2f} s timed region), {src}"


def run_workload(B, L, W, name, cfg_index, steps, warmup, phi_on, min_seconds=0.0, label=None):
    """Times `steps` passes of the whole hot path (rollout, Phi + tube, adjoint) over the device-resident workload W
    (or as many as fill `min_seconds`); returns the measurement block (value, per-kernel times, rooflines, clocks)."""
    torch = B.torch
    dev = B.dev
    batch, T, n, m = W.shape
    P = T * (T - 1) // 2
    _log(f"run_workload {label or name}: n={n} T={T} batch={batch} steps={steps} min_seconds={min_seconds}")
    d = {k: torch.from_numpy(getattr(W, k)).to(dev) for k in ("A", "B", "c", "x0", "u", "w", "g")}
    x = torch.empty((batch, T, n), device=dev)
    lam = torch.empty((batch, T, n), device=dev)
    gu = torch.empty((batch, T, m), device=dev)
    gx0 = torch.empty((batch, n), device=dev)
    if phi_on:
        phi = torch.empty((batch, P, n, n), device=dev)
        r = torch.empty((batch, T, n), device=dev)
        ws = torch.empty(max(16, L.ltv_scan_workspace_bytes(L.LTV_OP_SYSTEM_RESPONSE_TUBE, batch, T, n, 0)),
                         dtype=torch.uint8, device=dev)

    outs = dict(x=x, phi=phi, r=r, lam=lam, grad_u=gu, grad_x0=gx0) if phi_on else None
    fused = bool(phi_on and L.ltv_scan_all_is_fused(batch, T, n, m))

    def step():
        # the whole path in one call: ONE launch for small problems, else rollout + adjoint, then Phi + tube
        if phi_on:
            L.ltv_scan_all(d["A"], d["B"], d["c"], d["x0"], d["u"], d["w"], d["g"], outs=outs, workspace=ws)
        else:
            L.ltv_scan_rollout_adjoint(d["A"], d["B"], d["c"], d["x0"], d["u"], d["g"], x_out=x, lambda_out=lam,
                                       grad_u_out=gu, grad_x0_out=gx0)

    warm = max(warmup, 3)
    e0, e1 = _events(torch)
    B.barrier()
    e0.record()
    for _ in range(warm):
        step()
    e1.record()
    B.barrier()
    if min_seconds > 0:
        est = max(e0.elapsed_time(e1) / warm * 1e-3, 1e-6)
        steps = max(steps, int(min_seconds / est) + 1)
    L.ltv_profile_enable(True)
    l0 = L.ltv_launch_count()
    e0, e1 = _events(torch)
    B.barrier()
    t0 = time.time()
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    B.barrier()
    t1 = time.time()
    launches = L.ltv_launch_count() - l0
    prof = L.ltv_profile_collect()
    L.ltv_profile_enable(False)
    ms_total = B.max_over_ranks(e0.elapsed_time(e1))
    ms_step = ms_total / steps
    units = (P if phi_on else 1) * batch * B.world
    clocks = B.sampler.result(window=(t0, t1))
    out = dict(workload=label or name, n=n, m=m, T=T, batch_per_gpu=batch, steps=steps, warmup=warm,
               route=("ltv_scan_all: ONE fused launch per step (fused_small_kernel)" if fused else
                      "ltv_scan_all: rollout + adjoint, then Phi levels + tube" if phi_on else "ltv_scan_rollout_adjoint"),
               us_per_step=ms_step * 1e3,
               ms_per_step=ms_step, timed_region_s=ms_total * 1e-3,
               value=units / (ms_step * 1e-3), unit=UNIT if phi_on else UNIT_C5, gpu_launches=int(launches),
               kernel_ms_per_step={k: round(v[0] / steps, 5) for k, v in prof.items() if v[1]}, clocks=clocks)

    bytes_roll = batch * (T * (n * n + n * m + n + m) + n + T * n) * 4.0
    vec = {}
    for k in ("rollout", "adjoint"):
        if prof[k][1]:
            ms = prof[k][0] / prof[k][1]
            gbs = bytes_roll / (ms * 1e-3) / 1e9
            vec[k] = dict(per_s=batch * B.world / (ms * 1e-3), ms=ms, hbm_gbs=gbs, hbm_frac=gbs / B.pk["hbm_gbs"],
                          note="inside the concurrent pair: shares the SMs and HBM with the other scan")
    if prof["vector_pair"][1]:
        ms = prof["vector_pair"][0] / prof["vector_pair"][1]
        gbs = 2.0 * bytes_roll / (ms * 1e-3) / 1e9
        vec["pair"] = dict(per_s=batch * B.world / (ms * 1e-3), ms=ms, hbm_gbs=gbs, hbm_frac=gbs / B.pk["hbm_gbs"],
                           note="ltv_scan_rollout_adjoint: both scans side by side; bytes = rollout + adjoint (A read twice)")
    # each scan ALONE on the whole machine (the stand-alone calls), a few launches outside the timed step loop
    alone = {}
    for k, fn in (("rollout", lambda: L.ltv_scan_rollout(d["A"], d["B"], d["c"], d["x0"], d["u"], x_out=x)),
                  ("adjoint", lambda: L.ltv_scan_adjoint(d["A"], d["B"], d["g"], lambda_out=lam, grad_u_out=gu, grad_x0_out=gx0))):
        for _ in range(2):
            fn()
        a0, a1 = _events(torch)
        reps = 5
        B.barrier()
        a0.record()
        for _ in range(reps):
            fn()
        a1.record()
        B.barrier()
        ms = B.max_over_ranks(a0.elapsed_time(a1)) / reps
        gbs = bytes_roll / (ms * 1e-3) / 1e9
        alone[k] = dict(per_s=batch * B.world / (ms * 1e-3), ms=ms, hbm_gbs=gbs, hbm_frac=gbs / B.pk["hbm_gbs"])
    vec["alone"] = alone
    out["vector_scans"] = vec
    out["rollouts_per_s"] = vec.get("pair", {}).get("per_s")
    out["adjoints_per_s"] = vec.get("pair", {}).get("per_s")

    if phi_on and prof["phi_combine_tc"][1] > 0:
        G_blocks = (T - 1) * (T - 2) // 2                                   # GEMM blocks per item
        flops_issued = 3.0 * 2.0 * n ** 3 * G_blocks * batch                # 3xTF32, per step (all levels)
        ms_kernel = prof["phi_combine_tc"][0] / steps                       # all level launches of one step
        ach = flops_issued / (ms_kernel * 1e-3) / 1e12
        peak, src = B.tensor_peak(ms_total * 1e-3)
        clk = clocks["sm_mhz"] or 1965
        ceiling = 148 * 4096 * clk * 1e6 / 1e12            # 4096 dense tf32 flop / clk / SM at the sampled SM clock
        tr, tr_src = ncu_traffic(cfg_index, "phi_combine_tc") if label is None else (None, None)
        out["roofline"] = dict(
            bound="tensor", kernel="phi_combine_tc_kernel (3xTF32 tcgen05, all levels of one step)",
            achieved=ach, peak=peak, unit="TFLOP/s", frac=ach / peak, traffic=tr, traffic_source=tr_src,
            algorithmic="issued tf32 flop = 3 x 2 n^3 x (T-1)(T-2)/2 x batch per step (no padding, no split work)",
            peak_source=src, frac_of_unit_ceiling=ach / ceiling,
            unit_ceiling=f"{ceiling:.0f} TFLOP/s = 148 SM x 4096 flop/clk x {clk} MHz (median SM clock sampled in the timed region)",
            logical_fp32_tflops=ach / 3.0, kernel_ms_per_step=ms_kernel,
            launches_per_step=prof["phi_combine_tc"][1] / steps,
            share_of_step=ms_kernel / ms_step)
    elif fused:
        ms_f = prof["fused_small"][0] / max(prof["fused_small"][1], 1)
        # latency-bound by construction: the critical path is the chain of T-2 dependent n^3 products of column s = 0 on ONE SM
        chain_flop = 2.0 * n ** 3 * (T - 2)
        sm_peak = 128 * 2 * (clocks["sm_mhz"] or 1965) * 1e6          # fp32 FMA lanes of one SM
        out["roofline"] = dict(bound="alu", kernel="fused_small_kernel (critical path: column s = 0, one SM, fp32 FMA)",
                               achieved=chain_flop / (ms_f * 1e-3) / 1e9, peak=sm_peak / 1e9, unit="GFLOP/s (one SM)",
                               frac=chain_flop / (ms_f * 1e-3) / sm_peak, traffic=None, traffic_source=None,
                               algorithmic="2 n^3 (T-2) flop of the longest column chain over the kernel time; working set fits L2 / shared memory",
                               peak_source="128 fp32 FMA lanes x 2 flop x sampled SM clock (B300_MICROARCH.md unit counts)",
                               kernel_ms_per_step=ms_f, share_of_step=ms_f / ms_step)
    elif "pair" in vec:
        tr, tr_src = ncu_traffic(cfg_index, "vector_pair") if label is None else (None, None)
        out["roofline"] = dict(bound="hbm", kernel="rollout_kernel + adjoint_kernel running concurrently (ltv_scan_rollout_adjoint)",
                               achieved=vec["pair"]["hbm_gbs"],
                               peak=B.pk["hbm_gbs"], unit="GB/s", frac=vec["pair"]["hbm_frac"], traffic=tr,
                               traffic_source=tr_src,
                               algorithmic="bytes = 2 x batch x (T(n^2 + nm + n + m) + n + Tn) x 4 per step (each scan reads A once)",
                               peak_source=B.pk["source"] + " copy bandwidth (MEASURED_PEAKS.json hbm_gbs)",
                               kernel_ms_per_step=vec["pair"]["ms"], share_of_step=vec["pair"]["ms"] / ms_step)
    return out


def next_rows(B, L, W, steps):
    """SURVEY 8(f) rows, each timed alone on the device-resident C2 inputs (a few repetitions)."""
    torch, dev = B.torch, B.dev
    from workloads import observation_model

    batch, T, n, m = W.shape
    P = T * (T - 1) // 2
    p = 6
    d = {k: torch.from_numpy(getattr(W, k)).to(dev) for k in ("A", "B", "w")}
    out = {}

    def timed(fn, reps):
        for _ in range(2):
            fn()
        e0, e1 = _events(torch)
        B.barrier()
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        B.barrier()
        return B.max_over_ranks(e0.elapsed_time(e1)) / reps

    _log("next_rows: observer, kalman, constraints, output_feedback, output_feedback_constraints")
    gen = torch.Generator(device=dev).manual_seed(1234 + B.rank)
    Lt = torch.randn((batch, T, n, p), device=dev, generator=gen) * (0.05 / p ** 0.5)
    Cm = torch.randn((batch, T, p, n), device=dev, generator=gen) / n ** 0.5
    Kfb = torch.randn((batch, T, m, n), device=dev, generator=gen) * (0.2 / n ** 0.5)
    ff = torch.rand((batch, T, p), device=dev, generator=gen) * 4e-3 + 1e-3
    # NEXT-1: closed-loop observer propagation (14)
    nc = L.ltv_observer_row_floats(n, p)
    phio = torch.empty((batch, P, n, nc), device=dev)
    ro = torch.empty((batch, T, n), device=dev)
    wso = torch.empty(max(16, L.ltv_scan_workspace_bytes(L.LTV_OP_OBSERVER_RESPONSE, batch, T, n, p)), dtype=torch.uint8, device=dev)
    ms = timed(lambda: L.ltv_scan_observer_response(d["A"], Lt, Cm, d["w"], phi_out=phio, r_out=ro, workspace=wso), steps)
    out["observer"] = dict(p=p, ms=ms, blocks_per_s=batch * B.world * P / (ms * 1e-3),
                           issued_tf32_tflops=6.0 * n * n * nc * ((T - 1) * (T - 2) // 2) * batch / (ms * 1e-3) / 1e12)
    del phio, wso
    torch.cuda.empty_cache()
    # NEXT-3: Kalman recursion (13)
    Mobs = observation_model(batch, T, n, p, seed=777 + B.rank, kind="track")
    kd = [torch.from_numpy(Mobs[k]).to(dev) for k in ("C", "e", "f", "Pi0")]
    Lto = torch.empty((batch, T, n, p), device=dev)
    Pio = torch.empty((batch, T + 1, n, n), device=dev)
    wsk = torch.empty(max(16, L.ltv_scan_workspace_bytes(L.LTV_OP_KALMAN_GAINS, batch, T, n, p)), dtype=torch.uint8, device=dev)
    ms = timed(lambda: L.ltv_scan_kalman_gains(d["A"], *kd, Lt_out=Lto, Pi_out=Pio, workspace=wsk), steps)
    out["kalman"] = dict(p=p, ms=ms, recursions_per_s=batch * B.world / (ms * 1e-3),
                         issued_tf32_tflops=12.0 * n ** 3 * T * batch / (ms * 1e-3) / 1e12)
    del Pio, wsk, kd
    # NEXT-2: constraint margins (12d), open-loop form
    Hc = torch.randn((batch, T, 6, n), device=dev, generator=gen)
    sig = torch.empty((batch, T, 6), device=dev)
    wsc = torch.empty(max(16, L.ltv_scan_workspace_bytes(L.LTV_OP_CONSTRAINT_TIGHTENING, batch, T, n, 6)), dtype=torch.uint8, device=dev)
    ms = timed(lambda: L.ltv_scan_constraint_tightening(d["A"], d["w"], Hc, sigma_out=sig, workspace=wsc), steps)
    out["constraints"] = dict(nc=6, ms=ms, items_per_s=batch * B.world / (ms * 1e-3))
    del wsc
    # NEXT-4: assembled output-feedback responses (15) + tube (12e)
    #   default route (column recursion on D = Phi^xw - Phibar^x at this size) and the log-depth cross-scan route
    need = L.ltv_scan_workspace_bytes(L.LTV_OP_OUTPUT_FEEDBACK, batch, T, n, max(m, p))
    wsf = torch.empty(need, dtype=torch.uint8, device=dev)
    ms = timed(lambda: L.ltv_scan_output_feedback_response(d["A"], d["B"], Kfb, Lt, Cm, d["w"], ff, workspace=wsf), min(steps, 3))
    out["output_feedback"] = dict(p=p, ms=ms, blocks_per_s=batch * B.world * P / (ms * 1e-3), workspace_gb=need / 1e9)
    del wsf
    torch.cuda.empty_cache()
    L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, 1)
    try:
        need = L.ltv_scan_workspace_bytes(L.LTV_OP_OUTPUT_FEEDBACK, batch, T, n, max(m, p))
        wsf = torch.empty(need, dtype=torch.uint8, device=dev)
        ms1 = timed(lambda: L.ltv_scan_output_feedback_response(d["A"], d["B"], Kfb, Lt, Cm, d["w"], ff, workspace=wsf), min(steps, 3))
        out["output_feedback"].update(cross_scan_route_ms=ms1, cross_scan_route_workspace_gb=need / 1e9)
    finally:
        L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, 0)
    del wsf
    torch.cuda.empty_cache()
    # NEXT-4 / NEXT-2: input-side responses of (15) + closed-loop margins (12d), both terms, rows on [z; v]
    Hu = torch.randn((batch, T, 6, m), device=dev, generator=gen)
    wsq = torch.empty(L.lib.ltv_scan_output_feedback_constraints_workspace_bytes(batch, T, n, m, 6), dtype=torch.uint8, device=dev)
    ms = timed(lambda: L.ltv_scan_output_feedback_constraints(d["A"], d["B"], Kfb, Lt, Cm, d["w"], ff, Hc, Hu, workspace=wsq), steps)
    out["output_feedback_constraints"] = dict(p=p, nc=6, ms=ms, items_per_s=batch * B.world / (ms * 1e-3),
                                              note="Phi^uw, Phi^ue of (15) + sigma of (12d): backward sweep on the 2n-state closed loop")
    del wsq
    torch.cuda.empty_cache()
    # NEXT-4, general Phibar: eq.(15) + tube (12e) for a state-feedback response given as block operators (here: the
    # response of A + B Kfb and Kfb Phibar^x, produced on the device by the library's own Phi scan - input preparation,
    # outside the timed calls)
    Atil = d["A"] + torch.matmul(d["B"], Kfb)
    pbx, _ = L.ltv_scan_system_response_tube(Atil, d["w"])
    del Atil
    pbu = torch.zeros((batch, P + T, m, n), device=dev)
    wsa = torch.empty(L.lib.ltv_scan_output_feedback_assemble_workspace_bytes(batch, T, n, m, p), dtype=torch.uint8, device=dev)
    ms = timed(lambda: L.ltv_scan_output_feedback_assemble(d["A"], Lt, Cm, d["w"], ff, pbx, pbu, workspace=wsa), min(steps, 3))
    out["output_feedback_assemble"] = dict(p=p, ms=ms, blocks_per_s=batch * B.world * P / (ms * 1e-3),
                                           note="general Phibar: all four operators of (15) + tube, backward recursion over the columns "
                                                "(one n^3 product per block, T-1 batched tcgen05 GEMMs + fused row kernels)")
    # margins (12d), both terms, rows on [z; v], from the assembled operators of the general call
    asm = L.ltv_scan_output_feedback_assemble(d["A"], Lt, Cm, d["w"], ff, pbx, pbu, workspace=wsa)
    ms = timed(lambda: L.ltv_scan_operator_constraint_margins(asm["phi_xw"], Hc, d["w"], phi_uw=asm["phi_uw"], Hu=Hu,
                                                              phi_xe=asm["phi_xe"], phi_ue=asm["phi_ue"], f=ff), min(steps, 3))
    read_gb = batch * P * (n * n + m * n + n * p + m * p) * 4 / 1e9
    out["operator_constraint_margins"] = dict(nc=6, ms=ms, items_per_s=batch * B.world / (ms * 1e-3),
                                              hbm_gbs=read_gb / (ms * 1e-3), hbm_frac=read_gb / (ms * 1e-3) / B.pk["hbm_gbs"],
                                              note="eq.(12d) on assembled operators: every block read once")
    del asm, pbx, pbu, wsa
    torch.cuda.empty_cache()
    # the paper's own regime - ONE small problem (tens of states): the single-launch paths, in microseconds
    from workloads import dense_random
    small = {}
    for (ns, Ts) in ((40, 32), (64, 64)):
        Ws = dense_random(1, Ts, ns, 6, seed=ns + Ts, scale=0.3)
        Ms = observation_model(1, Ts, ns, p, seed=11, kind="track")
        As = torch.from_numpy(Ws.A).to(dev)
        ks = [torch.from_numpy(Ms[k]).to(dev) for k in ("C", "e", "f", "Pi0")]
        wsk = torch.empty(max(16, L.ltv_scan_workspace_bytes(L.LTV_OP_KALMAN_GAINS, 1, Ts, ns, p)), dtype=torch.uint8, device=dev)
        Lts = torch.empty((1, Ts, ns, p), device=dev)
        Pis = torch.empty((1, Ts + 1, ns, ns), device=dev)
        rec = timed(lambda: L.ltv_scan_kalman_gains(As, *ks, Lt_out=Lts, Pi_out=Pis, workspace=wsk), 20)
        scan = timed(lambda: L.ltv_scan_kalman_gains(As, *ks, Lt_out=Lts, Pi_out=Pis, workspace=wsk, mode=L.LTV_KALMAN_SCAN), 20)
        small[f"kalman_n{ns}_T{Ts}_batch1"] = dict(recursion_single_launch_us=rec * 1e3, riccati_scan_on_request_us=scan * 1e3)
    out["small_problem"] = small
    # SURVEY 8(e), optional: ONE large item split over GPUs by block rows (no data-path collective).  Measured on this one GPU
    # shard by shard (a rank's time is its own shard's; the multi-GPU time is the slowest shard), against the whole-item scan.
    from paper_2606_14188_b200.sharding import row_shard_range
    from workloads import config, generate
    del d
    torch.cuda.empty_cache()
    n4, T4 = 2400, 16                                       # one item of BASELINE.json configs[3]
    W4 = generate(config(3, batch=1))
    A4 = torch.from_numpy(W4.A).to(dev); w4 = torch.from_numpy(W4.w).to(dev)
    P4 = T4 * (T4 - 1) // 2
    phi4 = torch.empty((1, P4, n4, n4), device=dev); r4 = torch.empty((1, T4, n4), device=dev)
    ws4 = torch.empty(max(16, L.ltv_scan_workspace_bytes(L.LTV_OP_SYSTEM_RESPONSE_TUBE, 1, T4, n4, 0)), dtype=torch.uint8, device=dev)
    shards = dict(item="C4 item: n=2400 T=16 batch=1",
                  scan_whole_ms=timed(lambda: L.ltv_scan_system_response_tube(A4, w4, phi_out=phi4, r_out=r4, workspace=ws4), 3))
    del phi4
    for world in (1, 2, 4, 8):
        ts = []
        for rank in range(world):
            k_lo, k_hi = row_shard_range(T4, rank, world, n=n4)
            if k_hi <= k_lo:
                ts.append(0.0)
                continue
            po = torch.empty((1, L.ltv_phi_row_shard_blocks(T4, k_lo, k_hi), n4, n4), device=dev)
            ro = torch.zeros((1, T4, n4), device=dev)
            ts.append(timed(lambda: L.ltv_scan_system_response_tube_rows(A4, w4, k_lo, k_hi, phi_rows_out=po, r_out=ro), 3))
            del po
        shards[f"rows_{world}_shards_ms"] = [round(t, 3) for t in ts]
    shards["note"] = "each shard timed alone on this GPU; with one GPU per shard the item takes the slowest shard's time"
    out["row_shards"] = shards
    return out


def e2e_leg(B, L, W, phi_on, reps):
    """The same metric through ltv_scan_pipeline_host: pinned HOST buffers in, host results out, copies timed."""
    torch, dev = B.torch, B.dev
    batch, T, n, m = W.shape
    P = T * (T - 1) // 2
    units = (P if phi_on else 1) * batch * B.world
    _log("e2e leg (ltv_scan_pipeline_host)")
    need = L.ltv_scan_workspace_bytes(L.LTV_OP_PIPELINE_HOST if phi_on else L.LTV_OP_PIPELINE_HOST_NO_PHI, batch, T, n, m)
    wsh = torch.empty(need, dtype=torch.uint8, device=dev)
    h = {k: torch.from_numpy(getattr(W, k)).pin_memory() for k in ("A", "B", "c", "x0", "u", "w", "g")}
    if not phi_on:
        h.pop("w")
    h2d = sum(v.numel() * 4 for v in h.values())
    outs = None
    warm = 2                                   # the first calls also pay for page-locking effects and the copy stream's set-up
    times = []
    for i in range(warm + reps):
        B.barrier()
        t0 = time.perf_counter()
        outs = L.ltv_scan_pipeline_host(h["A"], h["B"], h["c"], h["x0"], h["u"], h["w"] if phi_on else None, h["g"],
                                        wsh, outs=outs)            # returns after the results are on the host (stream synchronised)
        if i >= warm:
            times.append(time.perf_counter() - t0)
    B.barrier()
    mean_sec = sum(times) / len(times)
    sec = B.max_over_ranks(sorted(times)[len(times) // 2])   # median step: a fresh box shows single outliers of 2x (mean / min / max beside it)
    d2h = sum(outs[k].numel() * 4 for k in ("x", "r", "lam", "grad_u", "grad_x0") if outs[k] is not None)
    del wsh
    torch.cuda.empty_cache()
    return dict(value=units / sec, unit=UNIT if phi_on else UNIT_C5, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
                ms_per_step=sec * 1e3, steps=reps, statistic="median of the timed steps", ms_mean=mean_sec * 1e3,
                ms_min=min(times) * 1e3, ms_max=max(times) * 1e3,
                note="ltv_scan_pipeline_host, pinned host buffers, upload of chunk i+1 overlapped with the compute of chunk i"
                     + ("; Phi (the largest result) stays in HBM where its consumers run: value counts x, r, lambda, "
                        "grad_u, grad_x0 back on the host" if phi_on else "; rollout + adjoint only"))


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist

    assert torch.cuda.is_available(), "bench.py needs a GPU (there is no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if args.tf32_peak:
        if rank == 0:
            print(json.dumps(dict(tf32_peak=measure_tf32_peak(torch.device("cuda", local), local))), flush=True)
        return
    import __graft_entry__ as G

    G.build()
    import paper_2606_14188_b200 as L
    from workloads import dense_random

    B = Bench(args, rank, world, local)
    full = args.config == 1 and not args.batch and not args.quick     # the default line carries every config
    if not args.no_tf32_peak:
        B.tf32 = measure_tf32_peak(B.dev, local, sustained_s=2.5)
        B.barrier()

    cfg, W = workload(args.config, rank, world, batch_override=args.batch or None)
    batch, T, n, m = W.shape
    P = T * (T - 1) // 2
    phi_on = args.config != 4
    head = run_workload(B, L, W, cfg["name"], args.config, args.steps, args.warmup, phi_on)

    sustained = dense = nxt = None
    others = {}
    if full or args.sustained:
        sustained = run_workload(B, L, W, cfg["name"], args.config, args.steps, args.warmup, phi_on, min_seconds=2.0)
    if full or args.next_rows:
        nxt = next_rows(B, L, W, max(3, min(args.steps, 10))) if phi_on else None
    e2e = None if args.no_e2e else e2e_leg(B, L, W, phi_on, args.e2e_steps)

    # ---- CPU oracle beside it (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        if args.cpu_items:
            items = min(batch, args.cpu_items)
        else:                                   # about 10-20 s of oracle work: calibrate on one item
            t1 = cpu_oracle_step(W, 1, phi_on)
            items = max(1, min(batch, int(12.0 / max(t1, 1e-3))))
        sec = cpu_oracle_step(W, items, phi_on)
        cpu = dict(value=items * (P if phi_on else 1) / sec, unit=UNIT if phi_on else UNIT_C5, cores=blas_threads(), kind="oracle",
                   sample=f"{items} of {batch} items of {cfg['name']}, whole path, fp64 numpy, {sec:.1f} s")

    if full:
        # the same shape on DENSE Jacobians (what PAPER.md:166 calls "dense matrix multiplications"): the like-for-like
        # figure against the library-GEMM peak, which is itself measured on dense random operands
        Wd = dense_random(batch, T, n, m, seed=4242 + rank)
        dense = run_workload(B, L, Wd, "dense_random", 1, args.steps, args.warmup, True, min_seconds=2.0,
                             label=f"dense random A_t = I + N(0, 0.5/sqrt(n)) at the C2 shape (n={n} T={T} batch={batch})")
        del Wd, W
        for ci, bo, st in ((0, None, 200), (2, None, 20), (3, None, 8), (4, 64, 40), (4, 256, 20), (4, 1024, 8)):
            c2, W2 = workload(ci, rank, world, batch_override=bo)
            key = f"C{ci + 1}" + (f"_b{bo}" if bo else "")
            others[key] = run_workload(B, L, W2, c2["name"], ci, st, 3, ci != 4)
            del W2

    B.sampler.stop_flag = True
    if rank == 0:
        a_gb = batch * T * n * n * 4 / 1e9
        phi_gb = batch * P * n * n * 4 / 1e9 if phi_on else 0.0
        line = dict(metric=METRIC, value=head["value"], unit=head["unit"], n_gpus=world,
                    steps=head["steps"], warmup=head["warmup"], ms_per_step=head["ms_per_step"], higher_is_better=True,
                    scaling="weak", vs_baseline=None, dtype="tf32x3/f32", data="synthetic",
                    config=dict(workload=f"{cfg['name']}: n={n} m={m} T={T} batch={batch} per GPU, "
                                         f"{P if phi_on else 0} Phi blocks/item (BASELINE.json configs[{args.config}])",
                                l2=(f"inputs (A {a_gb:.2f} GB) and outputs (Phi {phi_gb:.1f} GB) larger than the 126 MB L2; "
                                    "no flush" if a_gb > 0.3 else
                                    f"working set (A {a_gb * 1e3:.2f} MB) fits L2: warm-cache, latency-bound case"),
                                phi_layout="column-packed (LTV_PHI_COLUMN_PACKED, the scan's native order)"),
                    clocks=head["clocks"], e2e=e2e, gpu_launches=head["gpu_launches"], roofline=head.get("roofline"),
                    cpu_baseline=cpu, kernel_ms_per_step=head["kernel_ms_per_step"], vector_scans=head["vector_scans"],
                    rollouts_per_s=head["rollouts_per_s"], adjoints_per_s=head["adjoints_per_s"],
                    timed_region_s=head["timed_region_s"], tf32_peak=B.tf32, hbm_peak_gbs=B.pk["hbm_gbs"],
                    sustained=sustained, dense=dense, configs=others or None, next=nxt)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
