#!/usr/bin/env python
"""Benchmark of the per-patch Godunov hydro/MHD update (BASELINE.json metric: cell-updates/s and % of
the HBM roofline).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config5|config3_f32|config3_f64|config2|hydro_f32|hydro_ppm_f32|...]
  python bench.py --impl reference ...      # the CPU oracle on the host cores (the tier's reference arm)

A "step" is one pass of the whole hot path over the batch: amr_cfl_dt (O7, fused into the previous
step's epilogue; one 8-byte D->H read) and amr_mhd_step / amr_hydro_step (O0 halo assembly + O1..O6 +
the fused O7 of the new state).  Default workload: config 5 (512^3 cells as 4096 patches of 32^3, MHD,
fp32, MC + HLLD + GLM) -- the configuration the roofline target is quoted on; its synthetic initial
state is generated on the device (workloads.turbulence_patches_torch) and stands in for the paper's
cosmological run.  N > 1 runs N independent replicas, one per GPU (the path does not
shard: DESIGN.md §8), and reports the aggregate.

Prints ONE JSON line (rank 0).  Timing: CUDA events on the stream the library launches on, max over
ranks; --repeats regions (default 5) of exactly --steps steps each, the median region is reported; the
state (4.8 GB for config 5) is far larger than L2, so no flush is needed between steps.  Before any number
is printed one more step is compared with the oracle on 8 seeded patches (`parity`): a run that fails it
prints "value": null and exits 3.  The default run also times config 3 (256^3, fp32 and fp64) under `also`,
measures the plain FMA rate of the SMs for `alu_roofline.peak`, and times the oracle on all host cores and
on one core (`cpu_baseline`).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wk  # noqa: E402  (data only)

METRIC = "cell_updates_per_sec"
UNIT = "cell-updates/s"

# algorithmic bytes per cell-update: every interior value read once and written once
BYTES_PER_CELL = {("hydro", "f32"): 40, ("hydro", "f64"): 80, ("mhd", "f32"): 72, ("mhd", "f64"): 144}
# algorithmic floating-point operations per cell-update (add/sub/mul/min/max/abs/compare = 1,
# fma = 2, div and sqrt = 1; each face once, no halo recomputation), MC limiter, HLLC / HLLD+GLM
FLOPS_PER_CELL = {"hydro": 600, "mhd": 1700, "hydro_ppm": 1200}   # PPM: ~400 per cell and sweep (5 parabolas, tracing, HLLC), +-20 %


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), source="MEASURED_PEAKS.json (burst copy)", sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)))
    return dict(hbm_gbs=6650.0, source="fallback of B200_PROFILING.md", sm_max_mhz=1965.0)


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for nm, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        return dict(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), power_w_max=max(pw), samples=len(sm),
                    reasons=sorted(reasons))


def dram_traffic(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the step kernel on the full-size workload,
    from the committed ncu capture (profiles/*_dram_traffic.csv, newest round last); None if no capture exists
    for this workload (or the size was overridden)."""
    if workload is None:
        return None, None
    import csv, glob
    best = (None, None)
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_dram_traffic.csv"))):
        with open(path) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload:
                    best = (int(row["dram_bytes_read"]) + int(row["dram_bytes_write"]), row["source"])
    return best


def reduce_max_over_ranks(values, dist, device):
    """Replicas only: the one exchange of a multi-rank run.  Every timing of the job is the
    slowest rank's: element-wise MAX over ranks of a short list of floats (identity when dist is None)."""
    if dist is None:
        return [float(v) for v in values]
    import torch
    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def job_value(world: int, cells_per_rank: int, ms_per_step: float) -> float:
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's time."""
    return world * cells_per_rank / (ms_per_step * 1e-3)


def build_workload(name: str, device, size: int | None):
    """Returns dict(U=host pinned torch tensor [nf,np,n,n,n], origin, n, dx, domain, mhd, dtype, gamma, limiter,
    riemann, cfl, alpha, label)."""
    import torch
    if name == "config5":
        N = size or 512
        U, origin = wk.turbulence_patches_torch(N, 32, device)
        host = torch.empty(U.shape, dtype=torch.float32, pin_memory=torch.cuda.is_available())
        host.copy_(U)
        del U
        torch.cuda.empty_cache()
        return dict(U=host, origin=origin, n=32, dx=1.0 / N, domain=(N, N, N), mhd=True, dtype="f32", gamma=5.0 / 3.0,
                    limiter=wk.configs.LIM_MC, riemann=wk.configs.RS_HLLD, cfl=0.3, alpha=0.4,
                    label="config5: %d^3 cells, %d patches of 32^3 (+3 ghost in the API), MHD fp32, MC+HLLD+GLM" % (N, origin.shape[0]))
    if name in ("hydro_f32", "hydro_f64"):
        # not a BASELINE config: the config-5 field without B (rho = p = 1, Mach-3 turbulence), 32^3 patches, for the
        # hydro rows of the four-variant table in DESIGN.md section 7 (MC + HLLC)
        N = size or (512 if name.endswith("f32") else 256)
        U, origin = wk.turbulence_patches_torch(N, 32, device)
        U[4] -= 0.5 * (U[5] ** 2 + U[6] ** 2 + U[7] ** 2)
        dt = torch.float32 if name.endswith("f32") else torch.float64
        host = torch.empty((5,) + tuple(U.shape[1:]), dtype=dt, pin_memory=torch.cuda.is_available())
        host.copy_(U[:5])
        del U
        torch.cuda.empty_cache()
        return dict(U=host, origin=origin, n=32, dx=1.0 / N, domain=(N, N, N), mhd=False, dtype=name[-3:], gamma=5.0 / 3.0,
                    limiter=wk.configs.LIM_MC, riemann=wk.configs.RS_HLLC, cfl=0.3, alpha=0.0,
                    label="hydro: %d^3 cells, %d patches of 32^3, Mach-3 turbulence (config-5 recipe without B), hydro %s, MC+HLLC" % (N, origin.shape[0], name[-3:]))
    if name in ("hydro_ppm_f32", "hydro_ppm_f64"):
        # the next row of the scope table: the same gas as hydro_f32 (config-5 recipe without B,
        # Mach-1 here: PPM is run without CW84's optional flattening), advanced with the split PPM sweeps (HLLC)
        N = size or (512 if name.endswith("f32") else 256)
        U, origin = wk.turbulence_patches_torch(N, 32, device, mach=1.0)
        U[4] -= 0.5 * (U[5] ** 2 + U[6] ** 2 + U[7] ** 2)
        dt = torch.float32 if name.endswith("f32") else torch.float64
        host = torch.empty((5,) + tuple(U.shape[1:]), dtype=dt, pin_memory=torch.cuda.is_available())
        host.copy_(U[:5])
        del U
        torch.cuda.empty_cache()
        return dict(U=host, origin=origin, n=32, dx=1.0 / N, domain=(N, N, N), mhd=False, dtype=name[-3:], gamma=5.0 / 3.0,
                    limiter=wk.configs.LIM_MC, riemann=wk.configs.RS_HLLC, cfl=0.3, alpha=0.0, scheme="ppm",
                    label="hydro PPM: %d^3 cells, %d patches of 32^3, Mach-1 turbulence (config-5 recipe without B), hydro %s, PPM + HLLC, 3 sweeps per step" % (N, origin.shape[0], name[-3:]))
    if name in ("config3_f32", "config3_f64"):
        N = size or 256
        w = wk.config3_orszag_tang(N=N)
        lev = w.levels[0]
        dt = torch.float32 if name.endswith("f32") else torch.float64
        host = torch.empty(lev.U.shape, dtype=dt, pin_memory=torch.cuda.is_available())
        host.copy_(torch.from_numpy(lev.U))
        return dict(U=host, origin=lev.origin, n=16, dx=lev.dx, domain=lev.domain_cells, mhd=True, dtype=name[-3:],
                    gamma=w.gamma, limiter=w.limiter, riemann=w.riemann, cfl=w.cfl, alpha=w.alpha,
                    label="config3: %d^3 Orszag-Tang, %d patches of 16^3, MHD %s, MC+HLLD+GLM" % (N, lev.npatch, name[-3:]))
    if name == "config2":
        w = wk.config2_random_patches(npatch=size or 512)
        lev = w.levels[0]
        host = torch.empty(lev.U.shape, dtype=torch.float64, pin_memory=torch.cuda.is_available())
        host.copy_(torch.from_numpy(lev.U))
        return dict(U=host, origin=None, n=16, dx=lev.dx, domain=(16, 16, 16), mhd=False, dtype="f64", gamma=w.gamma,
                    limiter=w.limiter, riemann=w.riemann, cfl=w.cfl, alpha=0.0, self_periodic=True,
                    label="config2: %d self-periodic hydro patches of 16^3, fp64, MC+HLLC" % lev.npatch)
    raise SystemExit("unknown workload " + name)


def make_batch(W, device):
    import paper_1412_0934_b200 as amr
    nf, npatch = int(W["U"].shape[0]), int(W["U"].shape[1])
    dtype = amr.AMR_F32 if W["dtype"] == "f32" else amr.AMR_F64
    b = amr.PatchBatch(npatch, W["n"], nf, dtype, W["dx"], origin=W["origin"], domain_cells=W["domain"],
                       bc=(0,) * 6, self_periodic=bool(W.get("self_periodic", False)), nghost=3, device=str(device))
    return b


def one_step(b, W):
    dt, sm = b.cfl_dt(W["gamma"], W["cfl"])
    if W.get("scheme") == "ppm":
        W["_step_no"] = W.get("_step_no", 0) + 1
        b.hydro_step_ppm(dt, W["gamma"], W["riemann"], (W["_step_no"] - 1) % 2)
        return dt, sm
    if W["mhd"]:
        b.mhd_step(dt, W["gamma"], W["limiter"], W["riemann"], sm, W["alpha"])
    else:
        b.hydro_step(dt, W["gamma"], W["limiter"], W["riemann"])
    return dt, sm


def oracle_sample_level(W, npatch_sample: int):
    """First `npatch_sample` patches in Morton order (a contiguous cube of the domain), as their own periodic
    domain: a bounded sample of the same workload for the CPU oracle."""
    U = W["U"][:, :npatch_sample].numpy().astype(np.float64)
    n = W["n"]
    if W.get("self_periodic"):
        return wk.Level(n=n, g=3, level=0, dx=W["dx"], origin=np.zeros((npatch_sample, 3), np.int32),
                        domain_cells=(n, n, n), bc=(0,) * 6, self_periodic=True, U=U)
    origin = np.asarray(W["origin"][:npatch_sample])
    ext = origin.max(axis=0) + n
    assert int(np.prod(ext // n)) == npatch_sample, "sample must be a full Morton cube"
    return wk.Level(n=n, g=3, level=0, dx=W["dx"], origin=origin, domain_cells=tuple(int(v) for v in ext),
                    bc=(0,) * 6, self_periodic=False, U=U)


def oracle_time(W, npatch_sample: int, steps: int, warmup: int, threads: int | None = None):
    """Times the oracle, as it stands, on a bounded sample: `warmup` untimed steps, then `steps` timed ones.
    threads = None: all host cores (the OpenMP default)."""
    from oracle import api as oracle  # the cpu_baseline / reference legs may execute the oracle
    ncores = os.cpu_count() or 1
    oracle.set_num_threads(threads if threads else ncores)
    lev = oracle_sample_level(W, npatch_sample)
    wl = wk.Workload("sample", [lev], W["gamma"], W["mhd"], W["limiter"], W["riemann"], W["cfl"], 1, W["alpha"])
    times = []
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        oracle.advance(lev, wl, 1)
        if i >= warmup:
            times.append(time.perf_counter() - t0)
    used = oracle.num_threads()
    oracle.set_num_threads(ncores)
    return lev.ncells, times, used


def cpu_baseline_both(W, npatch: int):
    """BASELINE.md section 3 protocol: the oracle on all host cores AND on one core, one warm-up step and the
    median of three timed steps each, on bounded samples of the same workload (full Morton cubes of patches)."""
    big = 512 if npatch >= 512 else (64 if npatch >= 64 else (8 if npatch >= 8 else 1))
    small = 8 if W["n"] == 32 else min(big, 64)
    if W.get("self_periodic"):
        big, small = min(npatch, 512), min(npatch, 64)
    nc, t_all, threads = oracle_time(W, big, 3, 1)
    nc1, t_one, one = oracle_time(W, small, 3, 1, threads=1)
    m_all, m_one = statistics.median(t_all), statistics.median(t_one)
    return dict(value=nc / m_all, unit=UNIT, cores=threads, kind="oracle",
                sample="first %d patches in Morton order as a periodic sub-domain (%d cells), one warm-up + median of 3 steps "
                       "(O0+O7+O1..O6, fp64), %.2f s per step" % (big, nc, m_all),
                one_core=dict(value=nc1 / m_one, unit=UNIT, cores=one,
                              sample="first %d patches (%d cells), one warm-up + median of 3 steps, %.2f s per step" % (small, nc1, m_one)))


def parity_gate(b, W, nsample: int = 8):
    """parity is checked on the same run's output before any number is reported.  One more
    step is taken after the timed region; `nsample` seeded patches of its output are compared element by element
    with the oracle (the checker: fp64, same dt and c_h, the patch and its 26 neighbours cut out of the GPU's own
    input state; tests/gpu_harness.sampled_patch_parity, the routine of the full-size parity tests).  Tolerance:
    north_star's per-step bound (1e-12 fp64, 1e-5 fp32).  Outside every timed region."""
    tests_dir = os.path.join(ROOT, "tests")
    if tests_dir not in sys.path:
        sys.path.insert(0, tests_dir)
    import gpu_harness as H
    from oracle import api as oracle
    f32 = W["dtype"] == "f32"
    np_dtype = np.float32 if f32 else np.float64
    tol = 1e-5 if f32 else 1e-12
    U0 = b.download()
    dt, sm = one_step(b, W)
    U1 = b.download()
    npatch = int(U0.shape[1])
    rng = np.random.default_rng([wk.SEED, 2, npatch])
    ids = sorted(int(i) for i in rng.choice(npatch, size=min(nsample, npatch), replace=False))
    wl = dict(gamma=W["gamma"], limiter=W["limiter"], riemann=W["riemann"], alpha=W["alpha"])
    if W.get("scheme") == "ppm":
        # three sweeps with the ghost cells refilled before each: the whole 3x3x3 mini-level is swept (what enters
        # from beyond it travels 3 cells per sweep and never reaches the centre patch)
        order = oracle.PPM_ORDERS[(W["_step_no"] - 1) % 2]
        n = W["n"]
        where = {tuple(int(v) for v in o): i for i, o in enumerate(np.asarray(W["origin"]))}
        dom = np.asarray(W["domain"])
        mini = np.array([[i * n, j * n, k * n] for k in range(3) for j in range(3) for i in range(3)], np.int32)
        errs = []
        for s_ in ids:
            o = np.asarray(W["origin"][s_])
            sel = [where[tuple(int(v) for v in (o + (mo - n)) % dom)] for mo in mini]
            Ug = oracle.ghosted(np.ascontiguousarray(U0[:, sel]).astype(np.float64), 3)
            for d in order:
                oracle.fill_ghosts(Ug, 3, mini, (3 * n,) * 3, (0,) * 6, False)
                Ug = oracle.ppm_sweep(Ug, 3, d, dt, W["dx"], W["gamma"], W["riemann"])["U"]
            errs.append(H.rel_err(np.asarray(U1[:, s_:s_ + 1], np.float64), oracle.interior(Ug, 3)[:, 13:14]))
    elif W.get("self_periodic"):
        errs = []
        for s_ in ids:
            Um = np.ascontiguousarray(U0[:, s_:s_ + 1]).astype(np.float64)
            Ug = oracle.ghosted(Um, 3)
            oracle.fill_ghosts(Ug, 3, np.zeros((1, 3), np.int32), (W["n"],) * 3, (0,) * 6, True)
            r = oracle.step(Ug, 3, dt, W["dx"], W["gamma"], W["limiter"], W["riemann"], ch=sm, alpha=W["alpha"],
                            eps=oracle.default_eps(np_dtype))
            errs.append(H.rel_err(np.asarray(U1[:, s_:s_ + 1], np.float64), oracle.interior(r["U"], 3)))
    else:
        errs = H.sampled_patch_parity(oracle, U0, U1, W["origin"], W["n"], W["domain"], W["dx"], wl, dt, sm, ids, np_dtype)
    worst = float(max(float(e.max()) for e in errs))
    return dict(ok=bool(worst <= tol), max_rel_err=worst, tol=tol, patches=ids,
                how="one extra step after the timed region; %d seeded patches vs the fp64 oracle on their 3x3x3-patch neighbourhoods" % len(ids))


def timed_regions(b, W, K: int, repeats: int, dist, device):
    """`repeats` regions of EXACTLY K steps each, every region bracketed by barrier + synchronize, CUDA events on the
    library's stream; per-step events around the step call give the kernel time.  Returns (ms per step of each
    region, max over ranks; kernel ms of every step of every region, max over ranks)."""
    import torch
    regions, kernels = [], []
    for _ in range(repeats):
        ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
        ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
        start, end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        start.record()
        for i in range(K):
            dt, sm = b.cfl_dt(W["gamma"], W["cfl"])          # fused smax of the previous step: 8-byte D->H
            ev0[i].record()
            if W.get("scheme") == "ppm":
                W["_step_no"] = W.get("_step_no", 0) + 1
                b.hydro_step_ppm(dt, W["gamma"], W["riemann"], (W["_step_no"] - 1) % 2)
            elif W["mhd"]:
                b.mhd_step(dt, W["gamma"], W["limiter"], W["riemann"], sm, W["alpha"])
            else:
                b.hydro_step(dt, W["gamma"], W["limiter"], W["riemann"])
            ev1[i].record()
        end.record()
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        km = [a.elapsed_time(c) for a, c in zip(ev0, ev1)]
        vals = reduce_max_over_ranks([start.elapsed_time(end) / K] + km, dist, device)
        regions.append(vals[0])
        kernels.extend(vals[1:])
    return regions, kernels


def run_reference(args):
    """The tier's reference arm: the CPU oracle, as it stands, on the host cores, on a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    dev = torch.device("cuda:0") if torch.cuda.is_available() else torch.device("cpu")
    size = args.size
    if args.workload == "config5" and not torch.cuda.is_available():
        size = size or 128
    W = build_workload(args.workload, dev, size)
    npatch = int(W["U"].shape[1])
    sample = min(npatch, 64 if W["n"] == 32 else 512)
    ncells, times, threads = oracle_time(W, sample, args.steps, args.warmup)
    ms = 1e3 * sum(times) / len(times)
    value = ncells / (ms * 1e-3)
    kind = "mhd" if W["mhd"] else "hydro"
    out = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
               ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
               impl="reference",
               config=dict(workload=W["label"], physics=kind, sample="first %d patches in Morton order as a periodic sub-domain (%d cells) per step" % (sample, ncells)),
               cpu_baseline=dict(value=value, unit=UNIT, cores=threads, kind="oracle",
                                 sample="%d patches (%d cells), one O0+O7+O1..O6 step each" % (sample, ncells)),
               e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(out))


def run_builder(args):
    """--workload patch_builder: the next row of the scope table.  A step =
    amr_builder_build (Morton order + maximal compact cubic patches) + amr_builder_gather of every patch size,
    on the seeded refined-level workload (256^3 index space, ~25 % refined, 9 fp32 fields).  Same JSON contract;
    the metric counts cells built per second."""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    import paper_1412_0934_b200 as amr
    bits, kmax = args.size or 8, 5
    xyz, F = wk.refined_level_cells(bits)
    ncell, nf = xyz.shape[1], F.shape[0]
    hx = torch.from_numpy(xyz).pin_memory(); hf = torch.from_numpy(F).pin_memory()
    x, f = hx.cuda(), hf.cuda()
    b = amr.PatchBuilder(ncell)

    def step(xd, fd):
        b.build(xd, bits, kmax)
        outs = [b.gather(fd, k, want_origin=False)[0] for k in range(kmax + 1)]
        b.results(want_perm=False)          # patch table (first cell, level, origin) on the host
        return outs

    K, Wm = args.steps, max(args.warmup, 3)
    for _ in range(Wm):
        outs = step(x, f)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start(); time.sleep(0.25)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(K):
        outs = step(x, f)
    e1.record(); torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1) / K
    gathered = sum(int(o.shape[1]) * int(o.shape[2]) ** 3 for o in outs)
    assert gathered == ncell, "every cell belongs to exactly one patch"
    # end to end: cell list and fields from pinned host memory, patch arrays back to the host
    s2, t2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s2.record()
    for _ in range(3):
        outs = step(hx.cuda(non_blocking=True), hf.cuda(non_blocking=True))
        host = [o.cpu() for o in outs]
    t2.record(); torch.cuda.synchronize()
    ms2 = s2.elapsed_time(t2) / 3
    pk = peaks()
    bpc = 12 + 4 + 2 * nf * F.itemsize      # xyz in, curve order out, every field value read once and written once
    ach = bpc * ncell / (ms * 1e-3) / 1e9
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import patch_builder as pbo
        sx, sf = wk.refined_level_cells(bits - 1)
        t0 = time.perf_counter()
        perm, keys = pbo.curve_order(sx, bits - 1)
        first, level = pbo.build_patches(keys, kmax)
        for k in range(kmax + 1):
            pbo.gather_level(sf, perm, keys, first, level, k, bits - 1)
        dt = time.perf_counter() - t0
        cpu = dict(value=sx.shape[1] / dt, unit="cells/s", cores=1, kind="oracle",
                   sample="the same recipe at %d^3 (%d cells), build + gather of every level, %.1f s" % (1 << (bits - 1), sx.shape[1], dt))
    out = dict(metric="cells_built_per_sec", value=ncell / (ms * 1e-3), unit="cells/s", n_gpus=1, steps=K, warmup=Wm,
               ms_per_step=ms, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="u32", data="synthetic",
               config=dict(workload="patch_builder (f2): leaf cells of a refined level in a %d^3 index space, %d cells, %d fp32 fields, kmax=%d"
                           % (1 << bits, ncell, nf, kmax), step="amr_builder_build + amr_builder_gather for k = 0..%d" % kmax,
                           l2="working set %.0f MB; buffers alternate between sort passes" % (ncell * (16 + 2 * nf * 4) / 1e6)),
               roofline=dict(bound="hbm", achieved=ach, peak=pk["hbm_gbs"], unit="GB/s", frac=ach / pk["hbm_gbs"], traffic=None,
                             peak_source=pk["source"], kernel="sort passes + level + compaction + gather (whole step)",
                             kernel_ms=ms, bytes_per_cell=bpc),
               cpu_baseline=cpu,
               e2e=dict(value=ncell / (ms2 * 1e-3), unit="cells/s", h2d_bytes_per_step=int(xyz.nbytes + F.nbytes),
                        d2h_bytes_per_step=int(F.nbytes), ms_per_step=ms2, steps=3),
               gpu_launches=K * (1 + 3 * ((3 * bits + 7) // 8) + 6 + 3 * (kmax + 1) + 2 + (kmax + 1)), clocks=clocks, npatch=int(b.npatch))
    print(json.dumps(out))


def run_hierarchy(args):
    """--workload hierarchy3_f32 | hierarchy3_f64: the multi-level row of the scope table (
    PAPER.md:31, 59, 63).  A step = one root step of a three-level properly nested MHD hierarchy, all levels
    resident: amr_hierarchy_cfl_dt + amr_hierarchy_step (1 + 2 + 4 level steps with prolongation, restriction and
    reflux between them).  The metric counts cell-updates (cells of level l x 2^l per root step)."""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    import paper_1412_0934_b200 as amr
    f32 = args.workload.endswith("f32")
    nfine = args.size or 512
    wl = wk.config_hierarchy(True, 3, nfine, n=16)
    L = len(wl.levels)
    tdt = torch.float32 if f32 else torch.float64
    host = []
    for lv in wl.levels:
        h = torch.empty(lv.U.shape, dtype=tdt, pin_memory=torch.cuda.is_available())
        h.copy_(torch.from_numpy(lv.U))
        host.append(h)
    hier = amr.Hierarchy.from_workload(wl, amr.AMR_F32 if f32 else amr.AMR_F64)
    updates = sum(lv.ncells << l for l, lv in enumerate(wl.levels))

    def step():
        dt0, sm = hier.cfl_dt(wl.gamma, wl.cfl)
        hier.step(dt0, wl.gamma, wl.limiter, wl.riemann, sm, wl.alpha, True)

    K, Wm = args.steps, max(args.warmup, 3)
    for _ in range(Wm):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start(); time.sleep(0.25)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(K):
        step()
    e1.record(); torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1) / K
    # end to end: every level's state from pinned host memory, one root step, every level back
    nbytes = int(sum(h.numel() * h.element_size() for h in host))
    e2e = None
    if not args.no_e2e:
        for b, h in zip(hier.levels, host):
            b.upload(h.numpy())
        s2, t2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s2.record()
        for _ in range(3):
            for b, h in zip(hier.levels, host):
                b.upload(h.numpy())
            step()
            outs = [b.download() for b in hier.levels]
        t2.record(); torch.cuda.synchronize()
        ms2 = s2.elapsed_time(t2) / 3
        e2e = dict(value=updates / (ms2 * 1e-3), unit=UNIT, h2d_bytes_per_step=nbytes, d2h_bytes_per_step=nbytes,
                   ms_per_step=ms2, steps=3)
    # one regrid of the finest level between steps (amr_flag_blocks -> caller's selection -> new batch ->
    # amr_regrid_fill -> relink), wall-clock per part
    def new_level2():
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        l1 = wl.levels[1]
        flags = hier.levels[1].flag_blocks(0, 3.0)
        t1 = time.perf_counter()
        grid = wk.patch_flags_to_block_grid(l1, flags)
        cover1 = wk.origins_to_blocks(l1.origin, 16, wl.levels[0].domain_cells[0] // 8)
        origin_new = wk.blocks_to_origins(wk.select_blocks(grid, cover1, grow=False), 16)
        l2 = wl.levels[2]
        b2 = amr.PatchBatch(len(origin_new), 16, 9, amr.AMR_F32 if f32 else amr.AMR_F64, l2.dx, origin=origin_new,
                            domain_cells=l2.domain_cells, bc=(0,) * 6, self_periodic=False, nghost=3, level=2)
        t2 = time.perf_counter()
        b2.regrid_fill(hier.levels[2], hier.levels[1])
        torch.cuda.synchronize()
        return b2, origin_new, (t0, t1, t2, time.perf_counter())
    warm = new_level2()          # first use of the flag / copy / prolongation kernels and of the allocator: not timed
    b2, origin_new, (t0, t1, t2, t3) = new_level2()
    np_before = hier.levels[2].npatch
    hier.replace_level(2, warm[0])   # the same relink once, untimed (first touch of the link workspace)
    torch.cuda.synchronize()
    r0 = time.perf_counter()
    hier.replace_level(2, b2)
    torch.cuda.synchronize()
    r1 = time.perf_counter()
    step()
    torch.cuda.synchronize()
    regrid = dict(level=2, patches_before=int(np_before), patches_after=int(len(origin_new)), flag_ms=1e3 * (t1 - t0),
                  select_and_create_ms=1e3 * (t2 - t1), fill_ms=1e3 * (t3 - t2), relink_ms=1e3 * (r1 - r0),
                  note="wall clock, one regrid after the timed steps (the same regrid run once before, untimed, as warm-up); the block selection is host work (caller's policy), fill and link resolve cells on the device")
    pk = peaks()
    bpc = 2 * 9 * (4 if f32 else 8)
    ach = bpc * updates / (ms * 1e-3) / 1e9
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import api as oracle
        ws = wk.config_hierarchy(True, 3, 256, n=16)
        t0 = time.perf_counter()
        oracle.hierarchy_step(ws)
        dt = time.perf_counter() - t0
        nu = sum(lv.ncells << l for l, lv in enumerate(ws.levels))
        cpu = dict(value=nu / dt, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                   sample="the same recipe at 256^3 finest index space (%s; %d cell-updates), one root step, fp64, %.1f s" % (ws.note, nu, dt))
    # kernels per root step: level steps 2^l; per step of a level with a child: 2 prolongations, 1 restriction,
    # 1 reflux, 1 face-clear launch if it is a middle level; 1 smax launch per level whose fused smax was
    # invalidated by restriction / reflux
    launches = sum((1 << l) * (1 + (2 + 1 + 1 + (1 if l > 0 else 0) if l + 1 < L else 0)) for l in range(L)) + (L - 1)
    out = dict(metric=METRIC, value=updates / (ms * 1e-3), unit=UNIT, n_gpus=1, steps=K, warmup=Wm, ms_per_step=ms,
               higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32" if f32 else "f64", data="synthetic",
               config=dict(workload="hierarchy3 (f3): %d^3 finest index space, 16^3 patches, %s, MHD %s, MC+HLLD+GLM"
                           % (nfine, wl.note, "fp32" if f32 else "fp64"),
                           step="amr_hierarchy_cfl_dt + amr_hierarchy_step: 1 + 2 + 4 level steps, prolongation / restriction / reflux between levels",
                           cell_updates_per_step=updates,
                           l2="the whole hierarchy (%.0f MB) fits the 126 MB L2 only at small sizes; no flush: every level step rewrites its level" % (nbytes / 1e6)),
               roofline=dict(bound="hbm", achieved=ach, peak=pk["hbm_gbs"], unit="GB/s", frac=ach / pk["hbm_gbs"], traffic=None,
                             peak_source=pk["source"], kernel="whole root step (7 step-kernel launches + AMR operators)",
                             kernel_ms=ms, bytes_per_cell=bpc),
               cpu_baseline=cpu,
               e2e=e2e, gpu_launches=K * launches, clocks=clocks, regrid=regrid)
    print(json.dumps(out))


class _SoloTransport:
    """world = 1: nothing to exchange."""

    def exchange(self, rank, sendbuf, recvbuf):
        assert not sendbuf and not recvbuf

    @staticmethod
    def allreduce_max(v):
        return float(v)


def run_sharded(args):
    """--sharded: ONE level cut over the ranks instead of N replicas: config 3
    (256^3 Orszag-Tang, MHD; fp32 or fp64 by --workload config3_f32|config3_f64) or config 5 at --size, strong
    scaling.  Per step every rank refreshes its read-only copies (amr_patch_batch_export -> NCCL isend/irecv ->
    amr_patch_batch_import), all-reduces the signal speed and steps its owned patches.  With one GPU available only
    world = 1 could be run here; the exchange is covered by tests/test_sharding.py (gloo) and
    tests/test_gpu_sharding.py (emulated ranks, bitwise)."""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    import paper_1412_0934_b200 as amr
    from paper_1412_0934_b200 import sharding as sh
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    name = args.workload if args.workload.startswith("config3") else "config3_f32"
    f32 = name.endswith("f32")
    w = wk.config3_orszag_tang(N=args.size or 256)
    lev = w.levels[0]
    plan = sh.make_plans(lev.origin, lev.n, lev.domain_cells, lev.bc, world)[rank]
    shard = sh.ShardedBatch(plan, lev, amr.AMR_F32 if f32 else amr.AMR_F64, device=str(device))
    tr = sh.DistTransport(dist) if dist is not None else _SoloTransport()
    K, Wm = args.steps, args.warmup
    for _ in range(Wm):
        sh.sharded_step(shard, tr, w)
    regions = []
    for _ in range(max(1, args.repeats)):
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(K):
            sh.sharded_step(shard, tr, w)
        e1.record()
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        regions.append(reduce_max_over_ranks([e0.elapsed_time(e1) / K], dist, device)[0])
    ms = statistics.median(regions)
    nbytes = sum(len(v) for v in plan.send.values()) * lev.nfields * lev.n ** 3 * (4 if f32 else 8)
    if rank == 0:
        out = dict(metric=METRIC, value=lev.ncells / (ms * 1e-3), unit=UNIT, n_gpus=world, steps=K, warmup=Wm, repeats=len(regions),
                   ms_per_step=ms, higher_is_better=True, scaling="strong", vs_baseline=None, dtype="f32" if f32 else "f64", data="synthetic",
                   config=dict(workload="config3 sharded: %d^3 Orszag-Tang, %d patches of 16^3 cut into %d space-filling-curve ranges" % (lev.domain_cells[0], lev.npatch, world),
                               parallelism="one level sharded over %d GPU(s): halo copies + all-reduce(max) per step" % world,
                               halo_bytes_sent_per_step_rank0=int(nbytes), owned_patches_rank0=int(len(plan.owned)), copies_rank0=int(len(plan.ghost))),
                   gpu_launches=K * (1 + len(plan.send) + len(plan.recv)))
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config5")
    ap.add_argument("--size", type=int, default=None, help="override the grid size N (config3/5) or patch count (config2)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--repeats", type=int, default=5, help="timed regions of --steps steps each; the median is reported")
    ap.add_argument("--no-parity", action="store_true", help="skip the oracle parity gate (profiling runs only)")
    ap.add_argument("--no-also", action="store_true", help="skip the config-3 timings appended to the default run")
    ap.add_argument("--sharded", action="store_true", help="one level cut over the ranks (strong scaling) instead of replicas")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.sharded:
        if args.impl == "reference":
            raise SystemExit("the reference arm times the hot path on one host")
        return run_sharded(args)
    if args.workload == "patch_builder":
        if args.impl == "reference":
            raise SystemExit("the reference arm times the hot path (config 2, 3, 5); the patch builder's oracle is timed in cpu_baseline")
        return run_builder(args)
    if args.workload.startswith("hierarchy3"):
        if args.impl == "reference":
            raise SystemExit("the reference arm times the hot path (config 2, 3, 5); the hierarchy's oracle is timed in cpu_baseline")
        return run_hierarchy(args)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    import paper_1412_0934_b200 as amr  # fails loudly if libamrgodunov.so is missing

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)

    W = build_workload(args.workload, device, args.size)
    kind = "mhd" if W["mhd"] else "hydro"
    b = make_batch(W, device)
    b.upload(W["U"])
    ncells = b.ncells
    K, Wm, R = args.steps, args.warmup, max(1, args.repeats)

    for _ in range(Wm):
        one_step(b, W)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    regions, kern_ms = timed_regions(b, W, K, R, dist, device)
    clocks = sampler.stop() if rank == 0 else None
    ms_per_step = statistics.median(regions)          # median of the R regions of K steps each
    kern_med = statistics.median(kern_ms)
    value = job_value(world, ncells, ms_per_step)

    # validity of the evolved state, then parity of one more step against the oracle (the gate of SURVEY.md 8(d))
    counters = b.step_counters()
    tot = b.conserved_totals()
    state_ok = bool(np.all(np.isfinite(tot))) and counters["nonpositive_rho_after"] == 0
    parity = None
    if rank == 0 and not args.no_parity:
        parity = parity_gate(b, W)

    # end to end through the C-ABI with HOST buffers: H2D of the state, step, D2H of the new state
    e2e = None
    if not args.no_e2e:
        ke = min(K, 3)
        out_host = torch.empty(W["U"].shape, dtype=W["U"].dtype, pin_memory=torch.cuda.is_available())
        b.upload(W["U"]); one_step(b, W); b.download(out=out_host)   # warm
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        s2, e2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s2.record()
        for _ in range(ke):
            b.upload(W["U"])
            one_step(b, W)
            b.download(out=out_host)
        e2.record()
        torch.cuda.synchronize()
        ms2 = reduce_max_over_ranks([s2.elapsed_time(e2) / ke], dist, device)[0]
        nbytes = W["U"].numel() * W["U"].element_size()
        e2e = dict(value=job_value(world, ncells, ms2), unit=UNIT, h2d_bytes_per_step=int(nbytes),
                   d2h_bytes_per_step=int(nbytes + 8), ms_per_step=ms2, steps=ke)
        del out_host

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    pk = peaks()
    bpc = BYTES_PER_CELL[(kind, W["dtype"])]

    def roofline_of(kind_, dtype_, n_, ncells_, kms, workload_for_traffic):
        bpc_ = BYTES_PER_CELL[(kind_, dtype_)]
        kname = ("x2::godunov_step_x2_kernel" if dtype_ == "f32" else "d1::godunov_step_d1_kernel") if n_ % 16 == 0 else "godunov_step_kernel"
        if workload_for_traffic is not None and str(workload_for_traffic).startswith("hydro_ppm"):
            bpc_, kname = 3 * bpc_, "ppm::ppm_sweep_kernel (three launches per step: every value read and written once per sweep)"
        ach = bpc_ * ncells_ / (kms * 1e-3) / 1e9
        traffic, traffic_src = dram_traffic(workload_for_traffic)
        return dict(bound="hbm", achieved=ach, peak=pk["hbm_gbs"], unit="GB/s", frac=ach / pk["hbm_gbs"],
                    traffic=traffic, traffic_unit="bytes per launch (dram read + write, ncu --set full)",
                    traffic_source=traffic_src, peak_source=pk["source"], kernel=kname, kernel_ms=kms,
                    kernel_ms_how="median of the %d x %d per-step CUDA-event times" % (R, K),
                    bytes_per_cell=bpc_, frac_of_nominal_8TBs=ach / 8000.0)

    roof = roofline_of(kind, W["dtype"], W["n"], ncells, kern_med,
                       args.workload if (args.size is None or W.get("scheme") == "ppm") else None)
    # ALU roofline against the FMA rate MEASURED in this run (amr_measure_fma_peak: dependent-FMA chains on every SM)
    lanes = 128 if W["dtype"] == "f32" else 64
    nominal = 148 * lanes * pk["sm_max_mhz"] * 1e6 * 2 / 1e12          # TFLOP/s, fma = 2
    try:
        alu_peak = amr.measure_fma_peak(amr.AMR_F32 if W["dtype"] == "f32" else amr.AMR_F64, 2.0, str(device))
        alu_src = "measured in this run: amr_measure_fma_peak, ~2 ms of dependent-FMA chains on every SM"
    except Exception as exc:  # noqa: BLE001  (the bench line must still be printed)
        alu_peak, alu_src = nominal, "nominal (measurement failed: %s)" % exc
    fkind = "hydro_ppm" if W.get("scheme") == "ppm" else kind
    alu_ach = FLOPS_PER_CELL[fkind] * ncells / (kern_med * 1e-3) / 1e12
    alu = dict(bound="alu", achieved=alu_ach, peak=alu_peak, unit="TFLOP/s", frac=alu_ach / alu_peak,
               flops_per_cell=FLOPS_PER_CELL[fkind], peak_source=alu_src,
               nominal_peak=nominal, nominal_how="148 SMs x %d %s lanes x 2 (fma) x sm_max_mhz" % (lanes, W["dtype"]))

    # the 256^3 half of north_star's target, timed in the same run (not part of the headline value)
    also = None
    if args.workload == "config5" and args.size is None and world == 1 and not args.no_also:
        also = {}
        del b
        torch.cuda.empty_cache()
        for name in ("config3_f32", "config3_f64"):
            W3 = build_workload(name, device, None)
            b3 = make_batch(W3, device)
            b3.upload(W3["U"])
            for _ in range(3):
                one_step(b3, W3)
            reg3, k3 = timed_regions(b3, W3, 5, 3, None, device)
            p3 = None if args.no_parity else parity_gate(b3, W3)
            r3 = roofline_of("mhd", W3["dtype"], W3["n"], b3.ncells, statistics.median(k3), name)
            also[name] = dict(workload=W3["label"], cells=b3.ncells, steps=5, repeats=3, ms_per_step=statistics.median(reg3),
                              value=b3.ncells / (statistics.median(reg3) * 1e-3), unit=UNIT, kernel_ms=r3["kernel_ms"],
                              frac=r3["frac"], achieved_gbs=r3["achieved"], bytes_per_cell=r3["bytes_per_cell"],
                              traffic=r3["traffic"], parity=p3)
            del b3
            torch.cuda.empty_cache()

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_both(W, int(W["U"].shape[1]))

    parity_ok = None if parity is None else bool(parity["ok"] and all(v["parity"] is None or v["parity"]["ok"] for v in (also or {}).values()))
    out = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=Wm, repeats=R, ms_per_step=ms_per_step,
               ms_per_step_regions=regions, higher_is_better=True, scaling="weak", vs_baseline=None, dtype=W["dtype"], data="synthetic",
               config=dict(workload=W["label"], physics=kind, cells_per_gpu=ncells, l2="state %.2f GB per buffer >> 126 MB L2, no flush needed" % (ncells * bpc / 2 / 1e9),
                           parallelism="replicas only (no sharding)" if world > 1 else "single GPU",
                           step=("amr_cfl_dt (standalone smax reduction) + amr_hydro_step_ppm (x-y-z / z-y-x sweeps, alternating)" if W.get("scheme") == "ppm"
                                 else "amr_cfl_dt (fused smax, 8-byte D2H) + amr_%s_step" % kind),
                           timing="median of %d regions of exactly %d steps each (CUDA events, barrier + synchronize around every region)" % (R, K)),
               roofline=roof, alu_roofline=alu, also=also, cpu_baseline=cpu, e2e=e2e, gpu_launches=K, gpu_launches_all_regions=K * R,
               clocks=clocks, state_ok=state_ok, parity_ok=parity_ok, parity=parity, counters=counters)
    if parity_ok is False or not state_ok:
        # no number is reported from a run whose output fails parity (or went non-physical)
        out["value"] = None
        out["rejected"] = "parity gate failed" if parity_ok is False else "state went non-finite / non-positive"
        print(json.dumps(out))
        if dist is not None:
            dist.destroy_process_group()
        sys.exit(3)
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
