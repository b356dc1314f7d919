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
After the headline (configs[2]) the default run adds, each device-timed with its own clock record:
  configs        rows for configs[1], [3], [4] and the paper's own shapes (60^3 x 436, 80^3 x 901)
  config4_sweep  north_star's sweep: columns per rsdft_apply_h call = 32 ... 512 at configs[4]
  fft_sweep      the paper's Fig. 4 study (grid x batch 1 / 512) on the apply_h FFT kernels
  gemm_shapes    the paper's Fig. 2(b) shapes (K/N ~ 250, N = 2^p and 2^p +- 1) on the Gram and rotate kernels
  next1_eig, next2_rotate, next2_rotate2   the NEXT rows of SURVEY 8(f)
  library_yardstick  cuFFT / cuBLAS (through torch) on the same device data -- context, never on the library's path
N > 1: the path does not shard by contract ("no sharding, no collectives", BASELINE.json north_star;
DESIGN.md "Multi-GPU"): every rank runs an independent replica of the same block (weak scaling),
time = max over ranks, value = N * n * Ng / t.
--impl reference: the CPU oracle (oracle/) timed on the host cores on bounded samples of the same
workload (there is no reference implementation to install: /root/reference holds only the paper)."""
import argparse
import ctypes
import gc
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
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the rows beyond the headline (other configs, sweeps, shapes)")
    ap.add_argument("--batch", type=int, default=0, help="apply_h column batch width (0 = library default)")
    ap.add_argument("--streams", type=int, default=0, help="apply_h internal streams (0 = library default)")
    ap.add_argument("--ncol-per-call", type=int, default=0, help="columns per rsdft_apply_h call (config 4 sweep)")
    ap.add_argument("--pipeline", type=int, default=-1, help="apply_h FFT path: 0 three kernels per batch, 1 persistent pipeline kernel, 2 three kernels with the TMA x kernel (-1 = library default)")
    return ap.parse_args()


def workload_name(cfg_id):
    from paper_2512_04447_b200 import workloads as wl
    c = wl.CONFIGS[cfg_id]
    tag = "configs[%d]" % cfg_id if cfg_id <= 4 else "paper shape"
    return "%s %s: grid %d^3, L=%g bohr, %d atoms x %d KB projectors, m=%d, n=3m=%d columns" % (
        tag, c["name"], c["n"], c["L"], c["natom"], c["nproj"], c["m"], 3 * c["m"])


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
                kind_note="the long-double plain-loop oracle: a correctness tool, not a tuned CPU baseline",
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
            return self
        self.proc = subprocess.Popen([exe, "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits", "-lms", "100",
                                      "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()
        return self

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def mark(self):
        """number of samples taken so far (a row reports the samples that fell into its own timed region)"""
        return len(self.lines)

    @staticmethod
    def summarise(lines):
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in lines:
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

    def window(self, m0, m1=None):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        return self.summarise(self.lines[m0:m1])

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        return self.summarise(self.lines)


# ----------------------------------------------------------------------------- roofline denominators
def probe_peaks(sampler=None):
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_2512_04447_b200", "libpeakprobe.so"))
    out = {}
    v = ctypes.c_double()
    m0 = sampler.mark() if sampler else 0
    for kind, name in ((0, "dmma_tflops"), (1, "dfma_tflops")):
        rc = lib.peak_probe_fp64(kind, 150, ctypes.byref(v))            # ~0.4 s train: sustained figure
        if rc != 0:
            raise RuntimeError("peak_probe_fp64 failed: cudaError %d" % rc)
        out[name] = v.value
    rc = lib.peak_probe_copy(5, ctypes.byref(v))
    if rc != 0:
        raise RuntimeError("peak_probe_copy failed: cudaError %d" % rc)
    out["copy_gbs"] = v.value
    if sampler:
        time.sleep(0.15)
        out["clocks"] = sampler.window(m0)        # the probe's own clock record
    return out


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


GRAM_FLOPS_PER_CMAC = 6.0      # the kernel forms a complex multiply-add from 3 real MMAs (3M / Gauss form): 6 real flops, not 8
GRAM_TILE = 48


def gram_flops(n, ng, tile=GRAM_TILE):
    """(algorithmic, executed) REAL flops of one rsdft_subspace_gram launch: H in full + S upper triangle, 6 real flops per
    complex multiply-add (3M form; the conventional count is 8/6 of it); the executed count includes the padding of the
    last 48-column tile and the full diagonal tiles of S."""
    alg = GRAM_FLOPS_PER_CMAC * ng * (n * n + n * (n + 1) / 2.0)
    tm = (n + tile - 1) // tile
    return alg, GRAM_FLOPS_PER_CMAC * ng * tile * tile * (tm * tm + tm * (tm + 1) // 2)


def free_all():
    import torch
    gc.collect()
    torch.cuda.empty_cache()


# ----------------------------------------------------------------------------- one config, device-timed
def time_block_step(rsdft, wl, torch, cfg_id, steps, warmup, sampler, peaks, hbm_peak, per_call=0, args=None, keep=False, min_seconds=0.0):
    """apply_h + Gram on configs[cfg_id] with the block resident in HBM.  -> (row dict, state if keep)."""
    system = wl.make_system(cfg_id)
    ng = int(np.prod(system["n"]))
    m = system["m"]
    n = 3 * m
    plan = rsdft.plan_from_system(system)
    if args is not None:
        if args.batch:
            rsdft.rsdft_plan_set_batch(plan, args.batch)
        if args.streams:
            rsdft.rsdft_plan_set_streams(plan, args.streams)
        if args.pipeline >= 0:
            rsdft.rsdft_plan_set_pipeline(plan, args.pipeline)
    Y = wl.block_y(system, device="cuda")
    HY = torch.empty_like(Y)
    Hs = torch.empty((n, n), dtype=torch.complex128, device="cuda")
    Ss = torch.empty((n, n), dtype=torch.complex128, device="cuda")
    per_call = per_call if per_call > 0 else n
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

    t0 = time.perf_counter()
    for _ in range(max(warmup, 0)):
        step()
    torch.cuda.synchronize()
    if min_seconds > 0 and warmup > 0:          # launch-bound little configs: time enough steps for a clock record
        est = (time.perf_counter() - t0) / warmup
        steps = max(steps, min(2000, int(np.ceil(min_seconds / max(est, 1e-6)))))
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    launches[0] = 0
    m0 = sampler.mark() if sampler else 0
    t_begin = torch.cuda.Event(enable_timing=True)
    t_end = torch.cuda.Event(enable_timing=True)
    t_begin.record()
    for k in range(steps):
        step(evs[k])
    t_end.record()
    torch.cuda.synchronize()
    clocks = sampler.window(m0) if sampler else None
    total_ms = t_begin.elapsed_time(t_end)
    t_apply = float(np.mean([e[0].elapsed_time(e[1]) for e in evs])) * 1e-3
    t_gram = float(np.mean([e[1].elapsed_time(e[2]) for e in evs])) * 1e-3
    info = rsdft.rsdft_plan_info(plan)
    f_cov = info["sphere_points"] / ng
    bpp = 80.0 + 48.0 * f_cov                                      # SURVEY 8(d) design model
    alg, exe = gram_flops(n, ng)
    row = dict(workload=workload_name(cfg_id), steps=steps, warmup=warmup, ms_per_step=total_ms / steps, value=n * ng / (total_ms / steps * 1e-3),
               ms_apply_h=1e3 * t_apply, ms_gram=1e3 * t_gram, hx_pts_per_s=n * ng / t_apply,
               gram_tflops_executed=exe / t_gram / 1e12, gram_tflops_algorithmic=alg / t_gram / 1e12,
               gram_tflops_conventional=alg * 8.0 / GRAM_FLOPS_PER_CMAC / t_gram / 1e12,
               roofline_gram_frac=(alg / t_gram / 1e12 / peaks["dmma_tflops"]) if peaks else None,
               roofline_apply_h_frac=bpp * ng * n / t_apply / 1e9 / hbm_peak, apply_h_model_bytes_per_point=bpp,
               apply_h_floor_frac=32.0 * ng * n / t_apply / 1e9 / hbm_peak,
               ncol_per_apply_call=per_call, apply_batch_cols=info["batch_cols"], gpu_launches=launches[0], clocks=clocks)
    # cheap invariants on the timed results (full parity lives in tests/)
    Sd = torch.diagonal(Ss).real
    norms = (Y[:8].abs() ** 2).sum(dim=1)
    assert torch.allclose(Sd[:8], norms, rtol=1e-12), "S_sub diagonal disagrees with column norms"
    assert bool(torch.isfinite(torch.view_as_real(Hs)).all())
    if keep:
        return row, dict(system=system, plan=plan, Y=Y, HY=HY, Hs=Hs, Ss=Ss, ng=ng, m=m, n=n, t_apply=t_apply, t_gram=t_gram,
                         total_ms=total_ms, launches=launches[0], f_cov=f_cov)
    plan.close()
    del Y, HY, Hs, Ss
    free_all()
    return row, None


def timed(torch, fn, reps, warm=1):
    for _ in range(warm):
        fn()
    a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(reps):
        fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / reps * 1e-3


# ----------------------------------------------------------------------------- extras
def fft_sweep_rows(rsdft, wl, torch, sampler):
    """The paper's Fig. 4 study: time per wave function of the FFT Laplacian (plan without atoms:
    forward 3-D FFT, |G|^2/2, inverse 3-D FFT) for one orbital and for a batch of 512 (64 beyond 128^3)."""
    rows = []
    m0 = sampler.mark() if sampler else 0
    for N in (32, 48, 60, 64, 80, 96, 112, 128, 160, 192, 256):
        ng = N ** 3
        plan = rsdft.rsdft_plan_create((N, N, N), (0.2 * N,) * 3)
        for b in (1, 512 if N <= 128 else 64):
            X = wl.orbital_block(ng, range(min(b, 4)), 7, 0, device="cuda")
            if b > X.shape[0]:
                X = X.repeat((b + X.shape[0] - 1) // X.shape[0], 1)[:b].contiguous()
            HX = torch.empty_like(X)
            t = timed(torch, lambda: rsdft.rsdft_apply_h(plan, X, HX), 10 if b == 1 else 3, warm=2)
            rows.append(dict(grid=N, batch=b, us_per_wavefunction=1e6 * t / b, pts_per_s=b * ng / t,
                             nominal_fft_tflops=2 * 5.0 * ng * np.log2(ng) * b / t / 1e12))
            del X, HX
        plan.close()
        free_all()
    return dict(rows=rows, clocks=sampler.window(m0) if sampler else None,
                note="rsdft_apply_h without atoms, V_loc = 0; two 3-D transforms per wave function; nominal flops 2*5*Ng*log2(Ng)")


def gemm_shape_rows(rsdft, wl, torch, sampler, peaks):
    """The paper's rectangular GEMM study (Fig. 2(b): K/N = 250, N = 2^p and 2^p +- 1) on the Gram and
    rotate kernels: Y is K x N with K = the size of a plannable grid closest to 250 N (K/N = 256 at N = 2^p)."""
    rows = []
    m0 = sampler.mark() if sampler else 0
    for p2, grid in ((256, (16, 16, 256)), (512, (16, 32, 256)), (1024, (32, 32, 256)), (2048, (64, 32, 256))):
        K = int(np.prod(grid))
        plan = rsdft.rsdft_plan_create(grid, tuple(0.2 * g for g in grid))
        nmax = p2 + 1
        Y = wl.orbital_block(K, range(8), 3, 0, device="cuda").repeat((nmax + 7) // 8, 1)[:nmax].contiguous()
        HY = Y.roll(1, 0).contiguous()
        for N in (p2 - 1, p2, p2 + 1):
            Hs = torch.empty((N, N), dtype=torch.complex128, device="cuda")
            Ss = torch.empty((N, N), dtype=torch.complex128, device="cuda")
            t = timed(torch, lambda: rsdft.rsdft_subspace_gram(plan, Y[:N], HY[:N], Hs, Ss), 2)
            alg, exe = gram_flops(N, K)
            mrot = max(1, N // 3)
            Cm = Y[:mrot, :N].contiguous()
            Out = torch.empty((mrot, K), dtype=torch.complex128, device="cuda")
            tr = timed(torch, lambda: rsdft.rsdft_subspace_rotate(plan, Y[:N], Cm, Out), 2)
            rows.append(dict(N=N, K=K, K_over_N=K / N, gram_ms=1e3 * t, gram_tflops_algorithmic=alg / t / 1e12,
                             gram_tflops_executed=exe / t / 1e12, gram_frac_of_dmma_peak=alg / t / 1e12 / peaks["dmma_tflops"],
                             rotate_m=mrot, rotate_ms=1e3 * tr, rotate_tflops=GRAM_FLOPS_PER_CMAC * K * N * mrot / tr / 1e12,
                             rotate_tflops_conventional=8.0 * K * N * mrot / tr / 1e12))
            del Hs, Ss, Cm, Out
        plan.close()
        del Y, HY
        free_all()
    return dict(rows=rows, clocks=sampler.window(m0) if sampler else None,
                note="gram: [S|H] = Y^H [Y|HY], real flops 6*K*(N^2 + N(N+1)/2) algorithmic in the kernel's 3M form (executed counts the 48-column tile padding; "
                     "the conventional 8-flop count is 4/3 of it); "
                     "rotate: Out[K x N/3] = Y[K x N] C, real flops 6*K*N*m (3M form; conventional 8*K*N*m beside it)")


def library_yardstick(torch, st):
    """cuFFT and cuBLAS through torch on the same device data: context for the hand-written kernels, never on the
    library's own path.  FFT Laplacian of 19 columns (fftn, multiply, ifftn) and Y^H [Y | HY] as two ZGEMMs."""
    ng, n, Y, HY = st["ng"], st["n"], st["Y"], st["HY"]
    N = round(ng ** (1.0 / 3.0))
    out = {}
    try:
        nb = 19
        X = Y[:nb].reshape(nb, N, N, N)
        kin = torch.rand((N, N, N), dtype=torch.float64, device="cuda")
        t = timed(torch, lambda: torch.fft.ifftn(torch.fft.fftn(X, dim=(1, 2, 3)) * kin, dim=(1, 2, 3)), 3)
        out["cufft_laplacian_pts_per_s"] = nb * ng / t
        out["cufft_note"] = "torch.fft.fftn * table -> ifftn on %d columns (cuFFT + one elementwise pass; no V_loc, no projectors)" % nb
    except Exception as e:                                              # pragma: no cover
        out["cufft_error"] = str(e)[:200]
    try:
        ncols = min(n, 480)
        A = Y[:ncols]
        t = timed(torch, lambda: (A.conj() @ Y.T, A.conj() @ HY.T), 1)
        out["cublas_zgemm_tflops"] = 2 * 8.0 * ncols * n * ng / t / 1e12
        out["cublas_note"] = "torch.matmul (cuBLAS ZGEMM), %d x %d outputs of Y^H Y and Y^H HY over K = Ng (conj materialised by torch)" % (ncols, n)
    except Exception as e:                                              # pragma: no cover
        out["cublas_error"] = str(e)[:200]
    free_all()
    return out


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

    sampler = ClockSampler(local).start() if rank == 0 else None
    peaks = probe_peaks(sampler) if rank == 0 else None
    if world > 1:
        pk = torch.tensor([peaks["dmma_tflops"] if peaks else 0.0], dtype=torch.float64, device="cuda")
        dist.broadcast(pk, 0)
        if peaks is None:
            peaks = dict(dmma_tflops=float(pk.item()))
    mp = measured_peaks_file()
    hbm_peak = (mp or {}).get("hbm_gbs", 6650.0)

    # ---- headline: configs[args.config], block resident in HBM (seeded per column; every rank draws the same block)
    barrier()
    row, st = time_block_step(rsdft, wl, torch, args.config, args.steps, args.warmup, sampler, peaks, hbm_peak,
                              per_call=args.ncol_per_call, args=args, keep=True)
    barrier()
    plan, Y, HY, Hs, Ss, ng, m, n = st["plan"], st["Y"], st["HY"], st["Hs"], st["Ss"], st["ng"], st["m"], st["n"]
    ms_per_step = max_over_ranks(st["total_ms"]) / args.steps
    t_apply, t_gram = st["t_apply"], st["t_gram"]
    clocks = row["clocks"]

    # ---- the three FFT paths of rsdft_apply_h on the same block (informational; the headline ran the library default)
    paths = {}
    for mode, name in ((0, "three_kernels"), (1, "pipeline_kernel"), (2, "three_kernels_tma_x")):
        rsdft.rsdft_plan_set_pipeline(plan, mode)
        paths[name + "_ms"] = 1e3 * timed(torch, lambda: rsdft.rsdft_apply_h(plan, Y, HY), 2)
    rsdft.rsdft_plan_set_pipeline(plan, args.pipeline if args.pipeline >= 0 else 2)
    paths["note"] = ("rsdft_plan_set_pipeline 0 / 1 / 2 on the headline block, ms per apply_h call; bitwise identical results (tests); "
                     "the pipeline kernel keeps k-space in L2 (58 B of DRAM traffic per orbital*point against 112) but is bound by the "
                     "SM's L1/shared-memory data pipe, see DESIGN.md")

    # ---- optional Gram mode (H_sub from its upper tiles, mirrored): informational, not the headline
    rsdft.rsdft_plan_set_gram_mode(plan, 1)
    Hs2 = torch.empty_like(Hs)
    t_gram_hu = timed(torch, lambda: rsdft.rsdft_subspace_gram(plan, Y, HY, Hs2, Ss), 2)
    rsdft.rsdft_plan_set_gram_mode(plan, 0)
    dHu = float((Hs2 - Hs).abs().max() / Hs.abs().max())
    assert dHu <= 1e-13, "Hermitian-mode H_sub differs from the full contraction: %g" % dHu
    del Hs2

    # ---- NEXT-1: generalized eigen-solve of the (H_sub, S_sub) pencil just formed, both reductions
    eig = None
    lam = Cm = None
    try:
        rows_e = {}
        for mode, name in ((0, "trsm"), (1, "hegst")):
            rsdft.rsdft_plan_set_eig_mode(plan, mode, 0)
            lam, Cm = rsdft.rsdft_subspace_eig(plan, Hs, Ss, m)
            t0 = time.perf_counter()
            lam, Cm = rsdft.rsdft_subspace_eig(plan, Hs, Ss, m)
            torch.cuda.synchronize()
            wall = time.perf_counter() - t0
            s = rsdft.rsdft_subspace_eig_stats(plan)
            rows_e[name] = dict(ms_total=1e3 * wall, ms_potrf=s["ms_potrf"], ms_reduce=s["ms_reduce"], ms_eig=s["ms_eig"], ms_back=s["ms_back"],
                                jacobi_sweeps=int(s["sweeps"]), off_rel=s["off_rel"])
        rsdft.rsdft_plan_set_eig_mode(plan, 0, 0)
        lam, Cm = rsdft.rsdft_subspace_eig(plan, Hs, Ss, m)
        # validity of what was timed: residual and S-orthonormality on the device (C is n x m column-major in Cm[m, n])
        Hm, Sm, Cv = Hs.T, Ss.T, Cm.T
        res = float(((Hm @ Cv) - (Sm @ Cv) * lam).abs().max() / (Hm.abs().max() * Cv.abs().max() * n ** 0.5))
        orth = float((Cv.conj().T @ (Sm @ Cv) - torch.eye(m, dtype=torch.complex128, device="cuda")).abs().max())
        assert res <= 1e-11 and orth <= 1e-11, (res, orth)
        eig = dict(n=n, m=m, trsm=rows_e["trsm"], hegst=rows_e["hegst"],
                   reduce_hegst_over_trsm=rows_e["hegst"]["ms_reduce"] / rows_e["trsm"]["ms_reduce"],
                   residual_rel=res, orthonormality=orth,
                   note="rsdft_subspace_eig on the timed step's own (H_sub, S_sub): Cholesky, K = L^-1 H L^-H by two triangular solves "
                        "(PAPER.md eq. 1) or by the ZHEGST-style blocked reduction, block Jacobi on DMMA, back substitution; the paper "
                        "reports 1.5-2x from TRSM over HEGST on MI300A (PAPER.md:101)")
    except Exception as e:                                              # pragma: no cover
        eig = dict(error="%s: %s" % (type(e).__name__, str(e)[:300]))

    # ---- NEXT-2: the Rayleigh-Ritz update on the same block; informational
    rot = rot2 = None
    free_b, _ = torch.cuda.mem_get_info()
    if Cm is not None and "error" not in eig and free_b > (3 * m * ng * 16 + (4 << 30)):
        Xn = torch.empty((m, ng), dtype=torch.complex128, device="cuda")
        t_rot = timed(torch, lambda: rsdft.rsdft_subspace_rotate(plan, Y, Cm, Xn), 3)
        fl = GRAM_FLOPS_PER_CMAC * ng * n * m          # real flops of the 3M complex product (6 per complex multiply-add)
        rot = dict(ms=1e3 * t_rot, tflops=fl / t_rot / 1e12, frac_of_dmma_peak=fl / t_rot / 1e12 / peaks["dmma_tflops"],
                   conventional_8flop_tflops=fl * 8.0 / GRAM_FLOPS_PER_CMAC / t_rot / 1e12,
                   shape="Out[Ng x %d] = Y[Ng x %d] C[%d x %d]" % (m, n, n, m), note="rsdft_subspace_rotate, one call (X' = Y C_X); real flops 6*Ng*n*m (3M product)")
        HXn = torch.empty_like(Xn); R = torch.empty_like(Xn)
        t_rot2 = timed(torch, lambda: rsdft.rsdft_subspace_rotate2(plan, Y, HY, Cm, lam, Xn, HXn, R), 2)
        rnorm = float(R.abs().max() / HXn.abs().max())
        rot2 = dict(ms=1e3 * t_rot2, tflops=2 * fl / t_rot2 / 1e12, frac_of_dmma_peak=2 * fl / t_rot2 / 1e12 / peaks["dmma_tflops"],
                    conventional_8flop_tflops=2 * fl * 8.0 / GRAM_FLOPS_PER_CMAC / t_rot2 / 1e12,
                    max_abs_R_over_max_abs_HXnew=rnorm, algorithmic_bytes=(2 * n + 3 * m) * ng * 16,
                    note="rsdft_subspace_rotate2: X' = Y C, HX' = HY C, R = HX' - X' Lambda in one pass with the Ritz pairs of next1_eig; real flops 12*Ng*n*m (3M product) "
                         "(the block is random, so the residual is large: one Rayleigh-Ritz step of an unconverged LOBPCG)")
        del Xn, HXn, R

    yard = library_yardstick(torch, st) if (rank == 0 and not args.no_extras) else None

    # ---- end to end through the host-buffer entry point (N replicas, same max-over-ranks rule)
    e2e = None
    Hs_cpu, Ss_cpu = Hs.cpu(), Ss.cpu()
    hmax, smax = float(Hs.abs().max()), float(Ss.abs().max())
    gpu_launches = st["launches"]
    if not args.no_e2e:
        HY = None
        st["HY"] = None
        free_all()
        Yh = torch.empty((n, ng), dtype=torch.complex128, pin_memory=True)
        Yh.copy_(Y)
        Y = None
        st["Y"] = None
        free_all()
        Hh = torch.empty((n, n), dtype=torch.complex128, pin_memory=True)
        Sh = torch.empty((n, n), dtype=torch.complex128, pin_memory=True)
        rsdft.rsdft_block_step_host(plan, Yh, None, Hh, Sh)             # warm-up (allocates the plan's device block)
        barrier()
        a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.e2e_steps):
            rsdft.rsdft_block_step_host(plan, Yh, None, Hh, Sh)
        b.record()
        barrier()
        t_e2e = max_over_ranks(max(a.elapsed_time(b) * 1e-3, 0.0)) / args.e2e_steps
        # the host path contracts the Gram tiles panel by panel (other K split than the one-launch device path)
        dH = float((Hh - Hs_cpu).abs().max() / hmax)
        dS = float((Sh - Ss_cpu).abs().max() / smax)
        assert dH <= 1e-13 and dS <= 1e-13, "host path and device path disagree: %g %g" % (dH, dS)
        e2e = dict(value=world * n * ng / t_e2e, unit=UNIT, h2d_bytes_per_step=n * ng * 16, d2h_bytes_per_step=2 * n * n * 16,
                   ms_per_step=1e3 * t_e2e, steps=args.e2e_steps, api="rsdft_block_step_host (pinned host Y in, H_sub/S_sub out; H2D overlapped with apply_h and the panel-wise Gram)")
        del Yh, Hh, Sh
    plan.close()
    plan = Hs = Ss = Y = HY = lam = Cm = None
    st.clear()
    free_all()

    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return 0

    # ---- rows beyond the headline (rank 0, N = 1; each with its own clock record)
    extra = {}
    if not args.no_extras and world == 1:
        try:
            rows = {}
            for c in (0, 1, 3, 4, 5, 6):
                if c == args.config:
                    continue
                free_b, _ = torch.cuda.mem_get_info()
                cc = wl.CONFIGS[c]
                need = 2 * 3 * cc["m"] * cc["n"] ** 3 * 16 + (6 << 30)
                if free_b < need:
                    rows[str(c)] = dict(skipped="needs %.0f GB of free HBM, %.0f GB free" % (need / 1e9, free_b / 1e9))
                    continue
                r, _ = time_block_step(rsdft, wl, torch, c, 2, 1, sampler, peaks, hbm_peak, min_seconds=0.7)
                rows[str(c)] = r
            extra["configs"] = rows
            # north_star's sweep at configs[4]: columns per rsdft_apply_h call
            system = wl.make_system(4)
            ng4 = int(np.prod(system["n"])); n4 = 3 * system["m"]
            plan4 = rsdft.plan_from_system(system)
            Y4 = wl.block_y(system, device="cuda")
            HY4 = torch.empty_like(Y4)
            f4 = rsdft.rsdft_plan_info(plan4)["sphere_points"] / ng4
            sweep = []
            m0 = sampler.mark()
            for w in (32, 64, 128, 256, 512):
                def run(w=w):
                    for c0 in range(0, n4, w):
                        rsdft.rsdft_apply_h(plan4, Y4[c0:c0 + w], HY4[c0:c0 + w])
                t = timed(torch, run, 2)
                sweep.append(dict(ncol_per_call=w, ms_per_block=1e3 * t, hx_pts_per_s=n4 * ng4 / t,
                                  roofline_apply_h_frac=(80.0 + 48.0 * f4) * ng4 * n4 / t / 1e9 / hbm_peak))
            extra["config4_sweep"] = dict(rows=sweep, clocks=sampler.window(m0), workload=workload_name(4))
            plan4.close()
            del Y4, HY4
            free_all()
            extra["fft_sweep"] = fft_sweep_rows(rsdft, wl, torch, sampler)
            extra["gemm_shapes"] = gemm_shape_rows(rsdft, wl, torch, sampler, peaks)
        except Exception as e:                                          # pragma: no cover
            extra["extras_error"] = "%s: %s" % (type(e).__name__, str(e)[:300])

    # ---- roofline of the dominant kernel: gram_dmma_kernel (timed region = the rsdft_subspace_gram call:
    # one gram_dmma_kernel launch + one gram_reduce_kernel launch of ~0.1 % of its duration)
    flops_alg, flops_exec = gram_flops(n, ng)
    roofline = dict(bound="tensor", kernel="gram_dmma_kernel (FP64 DMMA.8x8x4, 3M complex product)", achieved=flops_alg / t_gram / 1e12,
                    peak=peaks["dmma_tflops"], unit="TFLOP/s", frac=flops_alg / t_gram / 1e12 / peaks["dmma_tflops"],
                    traffic=None,
                    traffic_source="not measured in this run (ncu cannot run inside the bench); the committed `ncu --set full` capture of this launch "
                                   "(profiles/r2_ncu_full_config2.md) read 632.7 GB of DRAM per launch = 15.5x the 40.8 GB operand floor (2*n*Ng*16 B), "
                                   "i.e. 1.23 TB/s = 15 % of the DRAM peak on a compute-bound kernel (48 x 48 tiles re-read the panels through L2)",
                    peak_source="libpeakprobe DMMA.8x8x4 register loop on this GPU, 150 launches back to back, clock record in peaks_probe.clocks "
                                "(MEASURED_PEAKS.json has no FP64 entry; bf16 %.1f TF x nominal 40/2250 = %.1f TF for context)" % (
                                    (mp or {}).get("bf16_tflops", float("nan")), (mp or {}).get("bf16_tflops", float("nan")) * 40 / 2250),
                    flops_per_launch=flops_alg, executed_flops_per_launch=flops_exec, executed_tflops=flops_exec / t_gram / 1e12,
                    ms_per_launch=1e3 * t_gram,
                    flops_definition="REAL flops the method needs in the kernel's 3M complex product (3 real MMAs = 6 flops per complex multiply-add, "
                                     "DESIGN.md 6.3): 6*Ng*(n^2 + n(n+1)/2) for H_sub in full + the upper triangle of S_sub; frac is the tensor-pipe view",
                    conventional_8flop_tflops=flops_alg * 8.0 / GRAM_FLOPS_PER_CMAC / t_gram / 1e12,
                    conventional_8flop_frac=flops_alg * 8.0 / GRAM_FLOPS_PER_CMAC / t_gram / 1e12 / peaks["dmma_tflops"])
    bpp = row["apply_h_model_bytes_per_point"]
    apply_roof = dict(bound="hbm", kernels="project/combine/fft3_fwd_zy/fft3_x/fft3_inv_yz/scatter (rsdft_apply_h)", achieved=bpp * ng * n / t_apply / 1e9,
                      peak=hbm_peak, peak_source="MEASURED_PEAKS.json hbm_gbs" if mp else "fallback 6650",
                      unit="GB/s", bytes_per_point=bpp, ms_per_call=1e3 * t_apply, probe_copy_gbs=peaks["copy_gbs"],
                      frac_of_32B_floor=row["apply_h_floor_frac"])
    apply_roof["frac"] = apply_roof["achieved"] / apply_roof["peak"]

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        cpu = oracle_sample(args.config)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "kind_note", "sample", "hx_pts_per_s", "gram_gflops")}
    all_clocks = sampler.stop() if sampler else None

    line = dict(metric=METRIC, value=world * n * ng / (ms_per_step * 1e-3), unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64 (complex128)",
                data="synthetic", config=dict(workload=workload_name(args.config), l2="inputs %.1f GB per block >> 126 MB L2, no flush needed" % (n * ng * 16 / 1e9),
                                              ncol_per_apply_call=row["ncol_per_apply_call"], apply_batch_cols=row["apply_batch_cols"], apply_streams=args.streams or 3,
                                              apply_fft_path={1: "persistent pipeline kernel (TMA tiles, L2-resident k-space)", 2: "three kernels per batch, TMA-staged x kernel"}.get(args.pipeline if args.pipeline >= 0 else 2, "three kernels per batch"), replicas=world),
                hx_pts_per_s=n * ng / t_apply, gram_tflops=flops_exec / t_gram / 1e12,
                gram_tflops_note="executed real FP64 flops / t (3M complex product: 6 flops per complex multiply-add; H_sub in full + upper tiles of "
                                 "S_sub, incl. tile padding); algorithmic (6*Ng*(n^2+n(n+1)/2)) = %.2f TF/s is roofline.achieved; in the conventional 8-flop "
                                 "count the same launch reads %.2f TF/s (roofline.conventional_8flop_tflops, above the DMMA peak because a quarter of the "
                                 "multiplies is never executed); the dense-equivalent 2*8*n^2*Ng count of SURVEY 8(d) would read %.2f TF/s and is NOT work done" % (
                                     flops_alg / t_gram / 1e12, flops_alg * 8.0 / GRAM_FLOPS_PER_CMAC / t_gram / 1e12, 16.0 * n * n * ng / t_gram / 1e12),
                ms_apply_h=1e3 * t_apply, ms_gram=1e3 * t_gram, roofline=roofline, roofline_apply_h=apply_roof,
                gram_hermitian_mode=dict(ms_gram=1e3 * t_gram_hu, ms_per_step=1e3 * (t_apply + t_gram_hu),
                                         value=world * n * ng / (t_apply + t_gram_hu), max_rel_diff_vs_full=dHu,
                                         note="rsdft_plan_set_gram_mode(1): H_sub upper tiles + conjugate mirror (30 % fewer flops). A production LOBPCG "
                                              "would run this mode (Hermitian eigen-solvers, rsdft_subspace_eig included, read one triangle); the headline keeps "
                                              "the full contraction because the definition and the paper's ZGEMM contract H_sub in full"),
                apply_h_paths=paths, next1_eig=eig, next2_rotate=rot, next2_rotate2=rot2,
                clocks=clocks, clocks_whole_run=all_clocks, e2e=e2e, gpu_launches=gpu_launches, cpu_baseline=cpu,
                peaks_probe=peaks, library_yardstick=yard)
    line.update(extra)
    print(json.dumps(line))
    return 0


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
