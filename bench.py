#!/usr/bin/env python
"""bench.py -- one LOBPCG block step (rsdft_apply_h on Y = [X, W, P], then rsdft_subspace_gram)
on a synthetic workload of BASELINE.json `configs`, timed on the device.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path over one block: HY = H Y for all
n = 3m columns, then H_sub = Y^H HY and S_sub = Y^H Y.  Prints ONE JSON line (rank 0).
  value      n*Ng / t_step        [orbital*grid-points/s]   inputs resident in HBM
  e2e        same, through rsdft_block_step_host with HOST (pinned) buffers, copies inside the timing
  gram_tflops, hx_pts_per_s       the two halves of BASELINE.json's metric, per call
  roofline   the dominant kernel (gram_dmma_kernel, FP64 tensor pipe), live CUDA-event timing
  cpu_baseline  the oracle as it stands on the host cores, bounded sample, extrapolated to the block
N > 1: the path does not shard by contract ("no sharding, no collectives", BASELINE.json north_star;
DESIGN.md "Multi-GPU"): every rank runs an independent replica of the same block (weak scaling),
time = max over ranks, value = N * n * Ng / t.
--impl reference: the CPU oracle (oracle/) timed on the host cores on bounded samples of the same
workload (there is no reference implementation to install: /root/reference holds only the paper)."""
import argparse
import ctypes
import json
import os
import shutil
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "H*X orbital-gridpoints/s through one LOBPCG block step (apply_h + Gram); Gram FP64 TFLOP/s"
UNIT = "orbital*gridpoints/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index (default 2: diamond-shaped)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--batch", type=int, default=0, help="apply_h column batch width (0 = library default)")
    ap.add_argument("--streams", type=int, default=0, help="apply_h internal streams (0 = library default)")
    ap.add_argument("--ncol-per-call", type=int, default=0, help="columns per rsdft_apply_h call (config 4 sweep)")
    ap.add_argument("--pipeline", type=int, default=-1, help="apply_h FFT path: 0 three kernels per batch, 1 persistent pipeline kernel (-1 = library default)")
    return ap.parse_args()


def workload_name(cfg_id):
    from paper_2512_04447_b200 import workloads as wl
    c = wl.CONFIGS[cfg_id]
    return "configs[%d] %s: grid %d^3, L=%g bohr, %d atoms x %d KB projectors, m=%d, n=3m=%d columns" % (
        cfg_id, c["name"], c["n"], c["L"], c["natom"], c["nproj"], c["m"], 3 * c["m"])


# ----------------------------------------------------------------------------- CPU oracle timing
def oracle_sample(cfg_id, ncols=None):
    """Times the oracle (as it stands) on a bounded sample of configs[cfg_id] and extrapolates to
    the full block.  -> dict(value, unit, cores, kind, sample, t_apply_per_col, gram_mac_per_s)."""
    from oracle import oracle
    from paper_2512_04447_b200 import workloads as wl
    cores = oracle.num_threads()
    system = wl.make_system(cfg_id)
    ng = int(np.prod(system["n"]))
    n = 3 * system["m"]
    ncols = cores if ncols is None else ncols
    X = wl.orbital_block(ng, range(ncols), system["seed"], 0).numpy()
    t0 = time.perf_counter()
    HX = oracle.apply_h(system, X)
    t_apply = time.perf_counter() - t0
    t0 = time.perf_counter()
    oracle.gram(X, HX)                          # ncols x ncols blocks of H_sub and S_sub over the full grid
    t_gram = time.perf_counter() - t0
    macs = 2.0 * ncols * ncols * ng             # complex multiply-adds done (H and S)
    rate_h = ncols * ng / t_apply               # orbital*points/s (includes building the sphere tables once)
    rate_g = macs / t_gram
    t_full = n * ng / rate_h + 2.0 * n * n * ng / rate_g
    return dict(value=n * ng / t_full, unit=UNIT, cores=cores, kind="oracle",
                sample="apply_h on %d of %d columns (%.1f s) + %dx%d blocks of H_sub,S_sub over the full grid (%.1f s); "
                       "extrapolated to n=%d (apply_h linear in n, Gram quadratic)" % (ncols, n, t_apply, ncols, ncols, t_gram, n),
                hx_pts_per_s=rate_h, gram_gflops=8.0 * rate_g / 1e9, t_sample_s=t_apply + t_gram)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    vals = []
    last = None
    for i in range(args.warmup + args.steps):
        last = oracle_sample(args.config, ncols=None)
        if i >= args.warmup:
            vals.append(last)
        if i == 0 and last["t_sample_s"] * (args.warmup + args.steps) > 240:      # keep the whole run to minutes
            vals = [last]
            break
    v = float(np.mean([x["value"] for x in vals]))
    n_ng = None
    from paper_2512_04447_b200 import workloads as wl
    c = wl.CONFIGS[args.config]
    n_ng = 3 * c["m"] * c["n"] ** 3
    line = dict(impl="reference", metric=METRIC, value=v, unit=UNIT, n_gpus=args.gpus, steps=len(vals), warmup=args.warmup,
                ms_per_step=1e3 * n_ng / v, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64 (long double accumulation)",
                data="synthetic", config=dict(workload=workload_name(args.config)),
                cpu_baseline=dict(value=v, unit=UNIT, cores=last["cores"], kind="oracle", sample=last["sample"]),
                e2e=dict(value=v, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        exe = shutil.which("nvidia-smi")
        if exe is None:
            return
        self.proc = subprocess.Popen([exe, "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits", "-lms", "100",
                                      "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for k, name in enumerate(names):
                if f[3 + k].lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)), samples=len(sm),
                    reasons=sorted(reasons))


# ----------------------------------------------------------------------------- roofline denominators
def probe_peaks():
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_2512_04447_b200", "libpeakprobe.so"))
    out = {}
    v = ctypes.c_double()
    for kind, name in ((0, "dmma_tflops"), (1, "dfma_tflops")):
        rc = lib.peak_probe_fp64(kind, 150, ctypes.byref(v))            # ~0.4 s train: sustained figure
        if rc != 0:
            raise RuntimeError("peak_probe_fp64 failed: cudaError %d" % rc)
        out[name] = v.value
    rc = lib.peak_probe_copy(5, ctypes.byref(v))
    if rc != 0:
        raise RuntimeError("peak_probe_copy failed: cudaError %d" % rc)
    out["copy_gbs"] = v.value
    return out


def ncu_traffic(cfg_id, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed
    `ncu --set full` capture of this config (profiles/ncu_traffic.csv), or None."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    try:
        for line in open(p).read().splitlines()[1:]:
            f = line.split(",")
            if int(f[0]) == cfg_id and f[1] == kernel:
                return float(f[2])
    except Exception:
        pass
    return None


def measured_peaks_file():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p))
        except Exception:
            return None
    return None


def max_over_ranks_value(x, world, device):
    """The timing rule of the multi-rank bench: every rank contributes its own device time, the job's time
    is the maximum (all_reduce MAX over the default process group; identity at world 1)."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# ----------------------------------------------------------------------------- the CUDA arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2512_04447_b200 import rsdft, workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback for the CUDA path")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    rsdft.load()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        return max_over_ranks_value(x, world, "cuda")

    cfg = wl.CONFIGS[args.config]
    system = wl.make_system(args.config)
    ng = int(np.prod(system["n"]))
    m = system["m"]
    n = 3 * m
    plan = rsdft.plan_from_system(system)
    if args.batch:
        rsdft.rsdft_plan_set_batch(plan, args.batch)
    if args.streams:
        rsdft.rsdft_plan_set_streams(plan, args.streams)
    if args.pipeline >= 0:
        rsdft.rsdft_plan_set_pipeline(plan, args.pipeline)
    peaks = probe_peaks() if rank == 0 else None

    # Y = [X, W, P] resident in HBM (seeded per column; every rank draws the same block)
    Y = wl.block_y(system, device="cuda")
    HY = torch.empty_like(Y)
    Hs = torch.empty((n, n), dtype=torch.complex128, device="cuda")
    Ss = torch.empty((n, n), dtype=torch.complex128, device="cuda")
    per_call = args.ncol_per_call if args.ncol_per_call > 0 else n

    launches = [0]

    def step(ev=None):
        if ev:
            ev[0].record()
        for c0 in range(0, n, per_call):
            rsdft.rsdft_apply_h(plan, Y[c0:c0 + per_call], HY[c0:c0 + per_call])
            launches[0] += rsdft.rsdft_plan_info(plan)["last_launches"]
        if ev:
            ev[1].record()
        rsdft.rsdft_subspace_gram(plan, Y, HY, Hs, Ss)
        launches[0] += rsdft.rsdft_plan_info(plan)["last_launches"]
        if ev:
            ev[2].record()

    for _ in range(max(args.warmup, 0)):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    launches[0] = 0
    barrier()
    t_begin = torch.cuda.Event(enable_timing=True)
    t_end = torch.cuda.Event(enable_timing=True)
    t_begin.record()
    for k in range(args.steps):
        step(evs[k])
    t_end.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = max_over_ranks(t_begin.elapsed_time(t_end))
    ms_per_step = total_ms / args.steps
    t_apply = float(np.mean([e[0].elapsed_time(e[1]) for e in evs])) * 1e-3
    t_gram = float(np.mean([e[1].elapsed_time(e[2]) for e in evs])) * 1e-3
    gpu_launches = launches[0]

    # sanity on the timed results (cheap invariants; full parity lives in tests/)
    Sd = torch.diagonal(Ss).real
    norms = (Y[:8].abs() ** 2).sum(dim=1)
    assert torch.allclose(Sd[:8], norms, rtol=1e-12), "S_sub diagonal disagrees with column norms"
    assert bool(torch.isfinite(torch.view_as_real(Hs)).all())

    # ---- optional Gram mode (H_sub from its upper tiles, mirrored): informational, not the headline
    rsdft.rsdft_plan_set_gram_mode(plan, 1)
    Hs2 = torch.empty_like(Hs)
    rsdft.rsdft_subspace_gram(plan, Y, HY, Hs2, Ss)
    g0 = torch.cuda.Event(enable_timing=True); g1 = torch.cuda.Event(enable_timing=True)
    g0.record()
    for _ in range(2):
        rsdft.rsdft_subspace_gram(plan, Y, HY, Hs2, Ss)
    g1.record()
    torch.cuda.synchronize()
    rsdft.rsdft_plan_set_gram_mode(plan, 0)
    t_gram_hu = g0.elapsed_time(g1) / 2 * 1e-3
    dHu = float((Hs2 - Hs).abs().max() / Hs.abs().max())
    assert dHu <= 1e-13, "Hermitian-mode H_sub differs from the full contraction: %g" % dHu
    del Hs2

    # ---- NEXT-2: the Rayleigh-Ritz update X' = Y C_X on the same block; informational
    rot = None
    free_b, _ = torch.cuda.mem_get_info()
    if free_b > (m * ng * 16 + (4 << 30)):
        Cx = wl.orbital_block(n, range(m), system["seed"], 7, device="cuda")       # [m, n]: column-major n x m
        Xn = torch.empty((m, ng), dtype=torch.complex128, device="cuda")
        rsdft.rsdft_subspace_rotate(plan, Y, Cx, Xn)
        r0 = torch.cuda.Event(enable_timing=True); r1 = torch.cuda.Event(enable_timing=True)
        r0.record()
        for _ in range(3):
            rsdft.rsdft_subspace_rotate(plan, Y, Cx, Xn)
        r1.record()
        torch.cuda.synchronize()
        t_rot = r0.elapsed_time(r1) / 3 * 1e-3
        rot = dict(ms=1e3 * t_rot, tflops=8.0 * ng * n * m / t_rot / 1e12,
                   frac_of_dmma_peak=(8.0 * ng * n * m / t_rot / 1e12 / peaks["dmma_tflops"]) if peaks else None, shape="Out[Ng x %d] = Y[Ng x %d] C[%d x %d]" % (m, n, n, m),
                   note="rsdft_subspace_rotate, one call (X' = Y C_X); flops 8*Ng*n*m")
        del Cx, Xn

    # ---- end to end through the host-buffer entry point (N replicas, same max-over-ranks rule)
    e2e = None
    if not args.no_e2e:
        del HY
        torch.cuda.empty_cache()
        Yh = torch.empty((n, ng), dtype=torch.complex128, pin_memory=True)
        Yh.copy_(Y)
        del Y
        torch.cuda.empty_cache()
        Hh = torch.empty((n, n), dtype=torch.complex128, pin_memory=True)
        Sh = torch.empty((n, n), dtype=torch.complex128, pin_memory=True)
        rsdft.rsdft_block_step_host(plan, Yh, None, Hh, Sh)             # warm-up (allocates the plan's device block)
        barrier()
        t0 = time.perf_counter()
        a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.e2e_steps):
            rsdft.rsdft_block_step_host(plan, Yh, None, Hh, Sh)
        b.record()
        barrier()
        t_e2e = max_over_ranks(max(a.elapsed_time(b) * 1e-3, 0.0)) / args.e2e_steps
        # the host path contracts the Gram tiles panel by panel (other K split than the one-launch device path)
        dH = float((Hh - Hs.cpu()).abs().max() / Hs.abs().max())
        dS = float((Sh - Ss.cpu()).abs().max() / Ss.abs().max())
        assert dH <= 1e-13 and dS <= 1e-13, "host path and device path disagree: %g %g" % (dH, dS)
        e2e = dict(value=world * n * ng / t_e2e, unit=UNIT, h2d_bytes_per_step=n * ng * 16, d2h_bytes_per_step=2 * n * n * 16,
                   ms_per_step=1e3 * t_e2e, steps=args.e2e_steps, api="rsdft_block_step_host (pinned host Y in, H_sub/S_sub out; H2D overlapped with apply_h and the panel-wise Gram)")

    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel: gram_dmma_kernel (timed region = the rsdft_subspace_gram call:
    # one gram_dmma_kernel launch + one gram_reduce_kernel launch of ~0.1 % of its duration)
    flops_alg = 8.0 * ng * (n * n + n * (n + 1) / 2.0)          # H full + S upper triangle
    tm = (n + 95) // 96
    flops_exec = 8.0 * ng * 96 * 96 * (tm * tm + tm * (tm + 1) // 2)
    mp = measured_peaks_file()
    roofline = dict(bound="tensor", kernel="gram_dmma_kernel (FP64 DMMA.8x8x4)", achieved=flops_alg / t_gram / 1e12,
                    peak=peaks["dmma_tflops"], unit="TFLOP/s", frac=flops_alg / t_gram / 1e12 / peaks["dmma_tflops"],
                    traffic=ncu_traffic(args.config, "gram_dmma_kernel"),
                    peak_source="libpeakprobe DMMA.8x8x4 register loop on this GPU, 150 launches back to back (MEASURED_PEAKS.json "
                                "has no FP64 entry; bf16 %.1f TF x nominal 40/2250 = %.1f TF for context)" % (
                                    (mp or {}).get("bf16_tflops", float("nan")), (mp or {}).get("bf16_tflops", float("nan")) * 40 / 2250),
                    flops_per_launch=flops_alg, executed_flops_per_launch=flops_exec, executed_tflops=flops_exec / t_gram / 1e12,
                    ms_per_launch=1e3 * t_gram)
    f_cov = rsdft.rsdft_plan_info(plan)["sphere_points"] / ng
    bytes_hx = (80.0 + 48.0 * f_cov) * ng * n                     # SURVEY 8(d) design model
    apply_roof = dict(bound="hbm", kernels="project/combine/fft3_fwd_zy/fft3_x/fft3_inv_yz/scatter (rsdft_apply_h)", achieved=bytes_hx / t_apply / 1e9,
                      peak=(mp or {}).get("hbm_gbs", 6650.0), peak_source="MEASURED_PEAKS.json hbm_gbs" if mp else "fallback 6650",
                      unit="GB/s", bytes_per_point=80.0 + 48.0 * f_cov, ms_per_call=1e3 * t_apply, probe_copy_gbs=peaks["copy_gbs"])
    apply_roof["frac"] = apply_roof["achieved"] / apply_roof["peak"]

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        cpu = oracle_sample(args.config)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "hx_pts_per_s", "gram_gflops")}

    line = dict(metric=METRIC, value=world * n * ng / (ms_per_step * 1e-3), unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64 (complex128)",
                data="synthetic", config=dict(workload=workload_name(args.config), l2="inputs %.1f GB per block >> 126 MB L2, no flush needed" % (n * ng * 16 / 1e9),
                                              ncol_per_apply_call=per_call, apply_batch_cols=rsdft.rsdft_plan_info(plan)["batch_cols"], apply_streams=args.streams or 3,
                                              replicas=world),
                hx_pts_per_s=n * ng / t_apply, gram_tflops=16.0 * n * n * ng / t_gram / 1e12,
                gram_tflops_note="nominal 2*8*n^2*Ng flops / t (SURVEY 8(d)); executed flops are in roofline.executed_tflops",
                ms_apply_h=1e3 * t_apply, ms_gram=1e3 * t_gram, roofline=roofline, roofline_apply_h=apply_roof,
                gram_hermitian_mode=dict(ms_gram=1e3 * t_gram_hu, ms_per_step=1e3 * (t_apply + t_gram_hu),
                                         value=world * n * ng / (t_apply + t_gram_hu), max_rel_diff_vs_full=dHu,
                                         note="rsdft_plan_set_gram_mode(1): H_sub upper tiles + conjugate mirror (30 % fewer flops); "
                                              "informational, the headline uses the full contraction"),
                next2_rotate=rot,
                clocks=clocks, e2e=e2e, gpu_launches=gpu_launches, cpu_baseline=cpu,
                peaks_probe=peaks)
    print(json.dumps(line))
    return 0


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
