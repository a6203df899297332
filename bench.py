#!/usr/bin/env python
"""bench.py -- coarse multi-RHS matvec + block-CG hot path on B200 (arXiv:2409.03904), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--nrhs S] [--config I]

A STEP is one pass of the whole hot path over one block of Nrhs synthetic
vectors: one BlockCGrQ iteration = stencil-GEMM apply Z = H D, Gram D^H Z, s x s algebra, the four block
rotations and the Gram T^H T (Fig. 2 left, statements 8-13), driven through the C ABI
(block_cg_begin / block_cg_step / block_cg_end).  Workload: BASELINE.json configs[3] -- the configuration
the metric "TFLOP/s & roofline fraction vs Nrhs" is quoted on (12^3 x 24 coarse lattice, 81-point stencil,
nbasis 32, complex64, ~27.5 GB of stencil matrices) -- at Nrhs = 16 unless --nrhs is given; the Nrhs sweep
1,4,8,16,32,64 of the apply kernel is reported under "sweep".  Inputs are seeded and synthetic
(DESIGN.md "Synthetic inputs"), resident in HBM before the timed region; the 27.5 GB operator is far larger
than L2, so no L2 flush is needed between iterations.

value      = algorithmic FLOP of K steps / device time (CUDA events, max over ranks), whole job, TFLOP/s
e2e        = same metric through block_cg_solve_host: pinned HOST buffers for B and X, H2D/D2H inside the timed region
roofline   = the dominant kernel (the stencil-GEMM apply) timed live with CUDA event pairs on its launch stream
cpu_baseline / --impl reference = the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from inputs import synth  # noqa: E402

METRIC = "coarse multi-RHS matvec TFLOP/s & roofline fraction vs Nrhs; block-CG solve s"      # BASELINE.json "metric"
METRIC_NOTE = ("value = algorithmic FLOP (8 per complex MAC) of one BlockCGrQ iteration (apply + 2 Gram + 4 rotations) / time; "
               "per-Nrhs apply TFLOP/s and roofline fractions under 'sweep'; solve seconds under 'block_cg_solve'")
UNIT = "TFLOP/s"
SM_COUNT, FP32_LANES, FP64_LANES = 148, 128, 64      # B200: guide's unit counts (blackwell_cuda_programming.md)
SWEEP = (1, 4, 8, 16, 32, 64)


# ---- algorithmic work (SURVEY.md section 8 / DESIGN.md "Algorithmic work") -----------------------------------
def apply_flops(V, nb, s):
    return 8.0 * 81 * V * nb * nb * s


def apply_bytes(V, nb, s, esize):
    return float(esize) * (81.0 * V * nb * nb + 2.0 * V * nb * s)          # A once, X once, Y once


def linalg_flops(V, nb, s):
    return 6.0 * 8.0 * V * nb * s * s                                        # 2 Gram products + 4 block rotations


def step_flops(V, nb, s):
    return apply_flops(V, nb, s) + linalg_flops(V, nb, s)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)),
                    bf16_tflops=float(p.get("bf16_tflops", 1590.0)),
                    bf16_tflops_sustained=float(p.get("bf16_tflops_sustained", p.get("bf16_tflops", 1400.0))), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0,
                source="fallback")                                           # B200_PROFILING.md fallback


def alu_peak_tflops(dtype, peaks):
    """FMA-pipe roof of the SIMT kernels: the MEASURED register-resident FFMA / DFMA rate of this device (coarse_measure_peaks),
    the nominal 148 SMs x lanes x 2 x max clock only if no measurement is at hand."""
    key = "ffma_tflops" if dtype == "c64" else "dfma_tflops"
    if peaks.get(key):
        return float(peaks[key])
    lanes = FP32_LANES if dtype == "c64" else FP64_LANES
    return SM_COUNT * lanes * 2.0 * peaks["sm_max_mhz"] * 1e6 / 1e12


def live_peaks(cm, peaks):
    """Adds the roofline denominators measured in this process on this device (the C-ABI bench helper coarse_measure_peaks):
    the HBM roof of the apply is a READ-ONLY stream (the operator is read once, never written); the copy figure of
    MEASURED_PEAKS.json stays beside it for context."""
    m = cm.measure_peaks()
    peaks = dict(peaks)
    peaks.update(hbm_copy_gbs=peaks["hbm_gbs"], hbm_gbs=max(float(m["hbm_read_gbs"]), peaks["hbm_gbs"]), hbm_read_gbs=float(m["hbm_read_gbs"]),
                 ffma_tflops=float(m["ffma_tflops"]), ffma2_tflops=float(m["ffma2_tflops"]), dfma_tflops=float(m["dfma_tflops"]),
                 dmma_tflops=float(m["dmma_tflops"]), hbm_peak_note="max(read-only stream measured live, copy figure of MEASURED_PEAKS.json)")
    return peaks


TF32_OVER_BF16 = 1.1 / 2.25     # nominal dense peaks (B200_PROFILING.md): the TF32 peak is the measured bf16 peak x this ratio
SPLIT_PRODUCTS = 3               # tensor-core products per algorithmic product (hi.hi + lo.hi + hi.lo, DESIGN.md 5.3 / 5.4)


def tensor_peak_tflops(peaks, sustained, kernel):
    """ALGORITHMIC TFLOP/s a split-precision tensor kernel could reach if the tensor pipe were the only limit:
    measured bf16 GEMM peak (sustained figure for a kernel timed inside a long step; binary16 runs at the bf16 rate)
    [x nominal TF32/bf16 ratio for the TF32 kernel] / 3 products."""
    bf16 = peaks["bf16_tflops_sustained"] if sustained else peaks["bf16_tflops"]
    ratio = TF32_OVER_BF16 if kernel.startswith("stencil_tc") else 1.0
    return bf16 * ratio / SPLIT_PRODUCTS


def roofline_tflops(V, nb, s, dtype, peaks, kernel="", sustained=True):
    """min(pipe peak, intensity x HBM bandwidth) for the apply; the pipe is the tensor pipe for the tcgen05 kernel
    (complex64, nrhs multiple of 8) and the FP32 / FP64 FMA pipe for the SIMT kernels."""
    esize = 8 if dtype == "c64" else 16
    intensity = apply_flops(V, nb, s) / apply_bytes(V, nb, s, esize)
    hbm = intensity * peaks["hbm_gbs"] / 1e3
    if kernel.startswith(("stencil_tc", "stencil_h16")):
        pipe, pipe_name = tensor_peak_tflops(peaks, sustained, kernel), "tensor"
    else:
        pipe, pipe_name = alu_peak_tflops(dtype, peaks), "alu"
    return dict(intensity=intensity, hbm_tflops=hbm, pipe_tflops=pipe, roof_tflops=min(hbm, pipe),
                bound="hbm" if hbm <= pipe else pipe_name)


# ---- clocks during the timed region (B200_PROFILING.md "clocks line") ----------------------------------------
class ClockSampler:
    """nvidia-smi in a loop beside the run.  It is started well BEFORE the timed region (its first line takes a few hundred ms, the
    timed region of the default run is under 200 ms) and every line carries a timestamp: stop(t0, t1) keeps the samples taken inside
    the timed region (host clock of the same box)."""
    FIELDS = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu, self.proc, self.path = gpu_index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self, t0=None, t1=None):
        """t0, t1: datetime.now() at the two ends of the timed region (None: every sample counts)"""
        from datetime import datetime, timedelta
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.proc is None:
            return out
        time.sleep(0.05)                                                   # let the sample of the last instants be written
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = []
        for line in open(self.path):
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                ts = datetime.strptime(f[0], "%Y/%m/%d %H:%M:%S.%f")
                rows.append((ts, float(f[1]), float(f[2]), {n for n, v in zip(names, f[5:9]) if v.lower().startswith("active")}))
            except ValueError:
                continue
        os.unlink(self.path)
        window = "timed region"
        pick = rows
        if t0 is not None and t1 is not None:
            pick = [r for r in rows if t0 <= r[0] <= t1]
            if not pick:                                                   # (a query takes 10-20 ms: the nearest samples around a very short region)
                pick = [r for r in rows if t0 - timedelta(seconds=0.1) <= r[0] <= t1 + timedelta(seconds=0.1)]
                window = "timed region +- 0.1 s"
        if pick:
            reasons = set().union(*[r[3] for r in pick])
            out.update(sm_mhz=float(np.median([r[1] for r in pick])), sm_max_mhz=float(np.max([r[2] for r in pick])), reasons=sorted(reasons),
                       samples=len(pick), window=window)
        return out


# ---- the CPU oracle on a bounded sample of the same workload ---------------------------------------------------
def oracle_sample_step(dims, nb, s, sites, A_s, X_full, K_small):
    """One 'step' of the oracle restricted to the sampled sites: apply on those sites (needs the whole X block for
    the neighbours), the two Gram products and the four block rotations on those sites' rows.  Returns seconds."""
    from oracle import oracle
    t0 = time.perf_counter()
    Z = oracle.apply(dims, A_s, X_full, sites=sites)                      # a2
    D = X_full[sites]
    G = oracle.gram(D, Z)                                                  # a3
    W = oracle.block_rotate(D, K_small, D, 1.0)                            # a5 (x4)
    T = oracle.block_rotate(Z, K_small, D, 1.0)
    G2 = oracle.gram(T, T)
    Q = oracle.block_rotate(T, K_small, T, 0.0)
    D2 = oracle.block_rotate(D, K_small, Q, 1.0)
    dt = time.perf_counter() - t0
    assert np.isfinite(G).all() and np.isfinite(G2).all() and np.isfinite(W).all() and np.isfinite(D2).all()
    return dt


def sample_sites(V, n, seed):
    rng = np.random.default_rng(seed)
    return np.sort(rng.choice(V, size=min(n, V), replace=False)).astype(np.int64)


def run_reference(args, cfg):
    """--impl reference: the oracle alone, on the box's host cores, each step a bounded sample of the workload."""
    from oracle import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    dims, nb, s = cfg["dims"], cfg["nbasis"], args.nrhs
    V = synth.volume(dims)
    n_sites = args.ref_sites
    sites = sample_sites(V, n_sites, 1)
    A_s = synth.stencil_matrices(dims, nb, cfg["seed"], sites)             # same seeded operator, sampled sites
    synth.add_shift(A_s, 90.0)                                             # representative diagonal shift (timing only)
    X = synth.make_block(dims, nb, s, cfg["seed"], synth.TAG_X)
    Ks = np.eye(s, dtype=np.complex128) * 0.5
    for _ in range(args.warmup):
        oracle_sample_step(dims, nb, s, sites[:max(1, n_sites // 8)], A_s[:max(1, n_sites // 8)], X, Ks)
    times = [oracle_sample_step(dims, nb, s, sites, A_s, X, Ks) for _ in range(args.steps)]
    total = float(np.sum(times))
    flops = step_flops(len(sites), nb, s) * args.steps
    value = flops / total / 1e12
    sample = f"{len(sites)} of {V} sites per step (apply on sampled sites with the full X block + Gram/rotations on their rows)"
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * total / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", impl="reference",
                config=dict(workload=cfg["name"], dims=list(dims), nbasis=nb, nrhs=s, storage="c64", sample=sample),
                cpu_baseline=dict(value=value, unit=UNIT, cores=oracle.num_threads(), kind="oracle", sample=sample),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))
    return 0


# ---- multi-rank plumbing (replicas only: DESIGN.md section 9) ---------------------------------------------------
def max_over_ranks(ms: float, world: int, device: str) -> float:
    """device time of the slowest rank (all_reduce MAX over the default process group)"""
    if world <= 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, steps: int, flops_per_step_per_rank: float, ms_max: float) -> float:
    """TFLOP/s of the whole job: every rank does the same work on its own replica (weak scaling)"""
    return world * steps * flops_per_step_per_rank / (ms_max * 1e-3) / 1e12


# ---- our arm ---------------------------------------------------------------------------------------------------
def time_apply(torch, op, X, Y, reps=20, warm=3):
    """ms per apply, `reps` launches back to back (CUDA events on the launch stream)"""
    for _ in range(warm):
        op.apply(X, Y)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    torch.cuda.synchronize()
    ev[0].record()
    for _ in range(reps):
        op.apply(X, Y)
    ev[1].record()
    torch.cuda.synchronize()
    return ev[0].elapsed_time(ev[1]) / reps


def next_rows_point(torch, cm, op, dims, nb, s, c, B, peaks):
    """SURVEY.md section 8(f) NEXT rows, measured (each is parity-tested in tests/): block project / promote at Table 6's shape
    (PAPER.md:570-571), multi-RHS deflation with 192 eigenvectors, the stacked and the preconditioned block solve on
    the bench operator.  Synthetic operands (random basis / eigenvector blocks: timing does not depend on their values)."""
    def timed(f, reps=10, warm=2):
        for _ in range(warm):
            f()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        for _ in range(reps):
            f()
        ev[1].record()
        torch.cuda.synchronize()
        return ev[0].elapsed_time(ev[1]) / reps
    rows = {}
    g = torch.Generator(device="cuda")
    g.manual_seed(20240903)
    Vc, vb, pnb, ps = 4096, 256, 64, 12
    Bas = torch.view_as_complex(torch.randn((Vc, vb, pnb, 2), device="cuda", generator=g))
    F = torch.view_as_complex(torch.randn((Vc, vb, ps, 2), device="cuda", generator=g))
    Cc = cm.block_project(Bas, F)
    by, fl = 8.0 * (Vc * vb * pnb + Vc * vb * ps + Vc * pnb * ps), 8.0 * Vc * vb * pnb * ps
    roof = min(peaks["hbm_gbs"] * 1e9 * fl / by, alu_peak_tflops("c64", peaks) * 1e12)
    for name, f in (("project", lambda: cm.block_project(Bas, F)), ("promote", lambda: cm.block_promote(Bas, Cc))):
        ms = timed(f)
        rows[name] = dict(shape="Vc 4096 x V_block 256 x nbasis 64 x nrhs 12, complex64 (Table 6)", ms=ms, gbs=by / ms / 1e6, tflops=fl / ms / 1e9,
                          frac_of_min_ffma_hbm=fl / (ms * 1e-3) / roof)
    del Bas, F, Cc
    n, nev = int(B.numel() // s), 192
    Vev = torch.view_as_complex(torch.randn((n, nev, 2), device="cuda", generator=g)) / float(np.sqrt(n))
    lam = [1.0 + i for i in range(nev)]
    ms = timed(lambda: op.deflate(Vev, lam, B), reps=5)
    rows["deflate"] = dict(shape=f"n {n} x nev {nev} x nrhs {s}, complex64", ms=ms, tflops=2 * 8.0 * n * nev * s / ms / 1e9,
                           gbs=8.0 * (2.0 * n * nev + 15.0 * n * s) / ms / 1e6)
    del Vev
    op.stacked_cg(B, tol=1e-6, maxiter=100)
    r = op.stacked_cg(B, tol=1e-6, maxiter=100)
    rows["stacked_cg"] = dict(seconds=r["seconds"], iterations=r["iterations"], status=r["status"], max_true_rel_res=max(r["rel_res_true"]))
    op.pblock_cg(B, lo=c - 12.0, hi=c + 12.0, order=8, tol=1e-6, maxiter=50)
    r = op.pblock_cg(B, lo=c - 12.0, hi=c + 12.0, order=8, tol=1e-6, maxiter=50)
    rows["pblock_cg_cheby8"] = dict(seconds=r["seconds"], iterations=r["iterations"], status=r["status"], max_true_rel_res=max(r["rel_res_true"]))
    return rows


def per_config_point(torch, cm, index, peaks):
    """One time-boxed apply + BlockCGrQ solve of another BASELINE.json configuration (parity-tested in tests/; reported here so
    that every figure quoted in DESIGN.md section 5 comes out of a tracked command)."""
    cfg = synth.config(index)
    dims, nb, s, dtype = cfg["dims"], cfg["nbasis"], cfg["nrhs"], cfg["dtype"]
    tdt = torch.complex64 if dtype == "c64" else torch.complex128
    esize = 8 if dtype == "c64" else 16
    V = synth.volume(dims)
    need = 81 * V * nb * nb * esize * 2.1 + 8 * V * nb * s * esize
    if torch.cuda.mem_get_info()[0] < need:
        return dict(config=index, workload=cfg["name"], skipped="not enough free device memory")
    A, c = cm.fill_synthetic(dims, nb, tdt, cfg["seed"], cfg["factor"])
    big = 81 * V * nb * nb * esize > 8 << 30
    op = cm.CoarseOperator(dims, A, s, flags=cm.binding.FLAG_TENSOR_ONLY if (big and dtype == "c64") else 0)
    del A
    torch.cuda.empty_cache()
    X = cm.fill_block(dims, nb, s, tdt, cfg["seed"], synth.TAG_X)
    Y = torch.empty_like(X)
    t_ms = time_apply(torch, op, X, Y, reps=20 if big else 100)
    kern = op.kernel_name(s)
    r = roofline_tflops(V, nb, s, dtype, peaks, kern, sustained=True)
    tf = apply_flops(V, nb, s) / (t_ms * 1e-3) / 1e12
    del Y
    B = cm.fill_block(dims, nb, s, tdt, cfg["seed"], synth.TAG_B)
    sol = op.block_cg(B, tol=cfg["tol"], maxiter=100, zero_guess=True)          # warm-up (kernel attributes, first touch)
    sol = op.block_cg(B, tol=cfg["tol"], maxiter=100, zero_guess=True)
    out = dict(config=index, workload=cfg["name"], dims=list(dims), nbasis=nb, nrhs=s, storage=dtype, kernel=kern,
               apply_ms=t_ms, apply_tflops=tf, apply_hbm_gbs=apply_bytes(V, nb, s, esize) / (t_ms * 1e-3) / 1e9,
               roof_tflops=r["roof_tflops"], bound=r["bound"], frac=tf / r["roof_tflops"],
               block_cg=dict(seconds=sol["seconds"], iterations=sol["iterations"], status=sol["status"], tol=cfg["tol"],
                             max_true_rel_res=max(sol["rel_res_true"])))
    op.close()
    del X, B, sol
    torch.cuda.empty_cache()
    return out


def load_traffic(key):
    """dram bytes per launch of the dominant kernel from the committed `ncu --set full` capture of this workload
    (key = workload|kernel@nrhs), or None when no capture of that combination is committed."""
    path = os.path.join(ROOT, "profiles", "apply_traffic.json")
    if os.path.exists(path):
        return json.load(open(path)).get(key)
    return None


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist

    import paper_2409_03904_b200 as cm

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    dims, nb, s, dtype = cfg["dims"], cfg["nbasis"], args.nrhs, cfg["dtype"]
    tdt = torch.complex64 if dtype == "c64" else torch.complex128
    esize = 8 if dtype == "c64" else 16
    V = synth.volume(dims)
    peaks = live_peaks(cm, measured_peaks())
    K, W = args.steps, args.warmup
    # replicas only: every rank holds the whole operator and iterates on its own block
    seed = cfg["seed"]
    clocks = ClockSampler(local_rank)                               # nvidia-smi beside the run from here on: its lines are time-stamped
    if rank == 0:
        clocks.start()
    A, c = cm.fill_synthetic(dims, nb, tdt, seed, cfg["factor"])
    nrhs_max = max(SWEEP) if (args.sweep and rank == 0) else s
    # nbasis 32 with wide blocks on the handle: keep both split-FP16 layouts (the kernel with the X operand in tensor memory is the
    # faster one above nrhs 48, the paired-site kernel below)
    flags = cm.binding.FLAG_H16X_WIDE if (nb == 32 and dtype == "c64" and nrhs_max > 48) else 0
    if dtype == "c64" and 81 * V * nb * nb * esize > (40 << 30) and nrhs_max >= 4:
        flags |= cm.binding.FLAG_TENSOR_ONLY                     # the 49 GB operator of configs[4]: one internal layout only
    op = cm.CoarseOperator(dims, A, nrhs_max, flags=flags)
    kernel_name = op.kernel_name(s)

    # bounded sample of canonical A for the oracle leg (inputs, read back before A is released)
    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        sites = sample_sites(V, args.cpu_sites, 1)
        A_s = A[torch.from_numpy(sites).cuda()].cpu().numpy()
    del A
    torch.cuda.empty_cache()

    B = cm.fill_block(dims, nb, s, tdt, seed + 1000 * rank, synth.TAG_B)
    X = torch.zeros_like(B)
    st, r0 = op.block_cg_begin(B, X, tol=1e-300)
    assert st == cm.binding.NOT_CONVERGED, st

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    op.block_cg_step(W)                                             # W untimed warm-up steps
    barrier()
    op.profile(True)
    l0 = cm.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    from datetime import datetime
    t_begin = datetime.now()
    e0.record()
    op.block_cg_step(K)                                             # exactly K timed steps
    e1.record()
    barrier()
    t_end = datetime.now()
    launches = cm.launch_count() - l0
    ms = e0.elapsed_time(e1)
    apply_ms = op.profile_read()
    op.profile(False)
    clk = clocks.stop(t_begin, t_end) if rank == 0 else None
    out = op.block_cg_end()
    assert out["status"] == 0, "block CG broke down inside the timed region"
    ms = max_over_ranks(ms, world, "cuda")
    value = whole_job_value(world, K, step_flops(V, nb, s), ms)

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    # ---- roofline object: the stencil-GEMM apply, timed per launch inside the timed region -----------------
    rf = roofline_tflops(V, nb, s, dtype, peaks, kernel_name, sustained=True)
    a_ms = float(np.mean(apply_ms)) if apply_ms else float("nan")
    a_tflops = apply_flops(V, nb, s) / (a_ms * 1e-3) / 1e12
    a_gbs = apply_bytes(V, nb, s, esize) / (a_ms * 1e-3) / 1e9
    # the same kernel, same block, 20 launches back to back (no linear algebra between them: the power-capped clock does not recover)
    Xb = cm.fill_block(dims, nb, s, tdt, seed, synth.TAG_X)
    Yb = torch.empty_like(Xb)
    bb_ms = time_apply(torch, op, Xb, Yb, reps=20)
    del Xb, Yb
    bb_tflops = apply_flops(V, nb, s) / (bb_ms * 1e-3) / 1e12
    bb_gbs = apply_bytes(V, nb, s, esize) / (bb_ms * 1e-3) / 1e9
    if rf["bound"] == "hbm":
        roofline = dict(bound="hbm", achieved=bb_gbs, peak=peaks["hbm_gbs"], unit="GB/s", frac=bb_gbs / peaks["hbm_gbs"],
                        frac_back_to_back=bb_gbs / peaks["hbm_gbs"], frac_in_step=a_gbs / peaks["hbm_gbs"],
                        peak_note=peaks.get("hbm_peak_note", "copy bandwidth of MEASURED_PEAKS.json"))
    else:
        roofline = dict(bound=rf["bound"], achieved=bb_tflops, peak=rf["pipe_tflops"], unit="TFLOP/s", frac=bb_tflops / rf["pipe_tflops"],
                        frac_back_to_back=bb_tflops / rf["pipe_tflops"], frac_in_step=a_tflops / rf["pipe_tflops"],
                        peak_note=("measured sustained bf16 GEMM [x nominal TF32/bf16 (1.1/2.25) for the TF32 kernel] / 3 products per algorithmic product"
                                   if rf["bound"] == "tensor" else "register-resident FMA loop measured on this device (coarse_measure_peaks)"))
    # a fraction well above 1 means the ceiling is wrong for this kernel (round 1 carried two ceilings): recorded in the line and on
    # stderr, not fatal -- the live stream figure moves by a few per cent from box to box and a dead bench reports nothing
    roofline["ceiling_check"] = "ok" if roofline["frac"] <= 1.08 else "frac above 1.08: the measured ceiling is too low for this kernel"
    if roofline["ceiling_check"] != "ok":
        print(f"bench.py: WARNING roofline {roofline['ceiling_check']}: {roofline}", file=sys.stderr)
    roofline.update(ms_per_launch_back_to_back=bb_ms, frac_note="frac = back to back (20 launches); frac_in_step = inside the timed BlockCGrQ steps",
                    traffic=load_traffic(f"{cfg['name']}|{kernel_name}@nrhs{s}"), kernel=kernel_name, launches_timed=len(apply_ms), ms_per_launch=a_ms,
                    share_of_step=a_ms * len(apply_ms) / ms if apply_ms else None, peak_source=peaks["source"],
                    intensity_flop_per_byte=rf["intensity"], hbm_gbs_achieved=a_gbs,
                    frac_of_min_peak_IxBW=a_tflops / rf["roof_tflops"])

    # ---- Nrhs sweep of the apply kernel (the metric's "vs Nrhs") --------------------------------------------
    sweep = []
    if args.sweep:
        for sv in SWEEP:
            Xs = cm.fill_block(dims, nb, sv, tdt, seed, synth.TAG_X)
            Ys = torch.empty_like(Xs)
            batches = [time_apply(torch, op, Xs, Ys, reps=20) for _ in range(2)]      # two batches of 20 launches back to back
            t_ms = min(batches)                                                        # (the power state of the board moves a batch by several %: the better one, both kept)
            r = roofline_tflops(V, nb, sv, dtype, peaks, op.kernel_name(sv), sustained=True)
            tf = apply_flops(V, nb, sv) / (t_ms * 1e-3) / 1e12
            # block-CG solve seconds at this Nrhs (the metric's second half): device-resident, X_0 = 0, to the config's tolerance
            Bs = cm.fill_block(dims, nb, sv, tdt, seed, synth.TAG_B)
            sol_s = op.block_cg(Bs, tol=cfg["tol"], maxiter=100, zero_guess=True)
            sweep.append(dict(nrhs=sv, ms=t_ms, tflops=tf, hbm_gbs=apply_bytes(V, nb, sv, esize) / (t_ms * 1e-3) / 1e9,
                              roof_tflops=r["roof_tflops"], bound=r["bound"], frac=tf / r["roof_tflops"],
                              kernel=op.kernel_name(sv), ms_batches=batches,
                              block_cg=dict(seconds=sol_s["seconds"], iterations=sol_s["iterations"], status=sol_s["status"],
                                            max_true_rel_res=max(sol_s["rel_res_true"]))))
            del Xs, Ys, Bs, sol_s

    # ---- block-CG solve seconds (the metric's second half), device-resident -----------------------------------
    Xs = torch.zeros_like(B)
    sol = op.block_cg(B, Xs, tol=cfg["tol"], maxiter=100)
    bcg = dict(seconds=sol["seconds"], iterations=sol["iterations"], status=sol["status"], tol=cfg["tol"],
               max_true_rel_res=max(sol["rel_res_true"]))

    # ---- Chebyshev polynomial coarse solve (the paper's coarse solve is order 120) ----
    cheb = None
    if args.cheby_order > 0:
        lo_c, hi_c = c - 12.0, c + 12.0                 # safely around the synthetic operator's spectrum (c +- 7)
        op.cheby_apply(B, lo_c, hi_c, 3, X=Xs)          # warm-up
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        op.cheby_apply(B, lo_c, hi_c, args.cheby_order, X=Xs)
        ev[1].record()
        torch.cuda.synchronize()
        t_c = ev[0].elapsed_time(ev[1]) * 1e-3
        napp = args.cheby_order - 1
        # the polynomial's residual bound on a spectrum inside [lo, hi]:  ||B - H X|| / ||B|| <= 1 / |T_n(y(0))|  (
        # closed form pinned in tests/test_oracle_cheby.py), evaluated with one more apply
        Yc = op.apply(Xs)
        res_c = float((torch.linalg.vector_norm((B - Yc).reshape(-1, s), dim=0) / torch.linalg.vector_norm(B.reshape(-1, s), dim=0)).max())
        y0 = (hi_c + lo_c) / (hi_c - lo_c)
        bound_c = 1.0 / np.cosh(args.cheby_order * np.arccosh(y0))
        del Yc
        assert res_c <= bound_c + 5e-6, ("Chebyshev solve misses its residual bound", res_c, bound_c)
        cheb = dict(order=args.cheby_order, lo=lo_c, hi=hi_c, seconds=t_c, applies=napp,
                    tflops=napp * apply_flops(V, nb, s) / t_c / 1e12, max_rel_res=res_c, residual_bound=float(bound_c),
                    vs_applies_only=t_c / (napp * bb_ms * 1e-3))

    # ---- e2e: the same solve through the C-ABI call with pinned HOST buffers ----------------------------------
    # X_0 = 0 (the workload's initial guess): COARSE_SOLVE_ZERO_GUESS -- B host->device, solve, X device->host
    Bh = B.cpu().pin_memory()
    Xh = torch.empty_like(Bh).pin_memory()
    op.block_cg_host(Bh, Xh, tol=cfg["tol"], maxiter=100, zero_guess=True)      # warm-up
    Xh.fill_(float("nan"))
    l1 = cm.launch_count()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    sol_h = op.block_cg_host(Bh, Xh, tol=cfg["tol"], maxiter=100, zero_guess=True)
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    assert sol_h["status"] == 0 and bool(torch.isfinite(torch.view_as_real(Xh)).all())
    its = sol_h["iterations"]
    fl_e2e = (its + 1) * apply_flops(V, nb, s) + its * linalg_flops(V, nb, s) + 3 * 8.0 * V * nb * s * s
    blk_bytes = V * nb * s * esize
    e2e = dict(value=fl_e2e / t_e2e / 1e12, unit=UNIT, h2d_bytes_per_step=blk_bytes / max(its, 1),
               d2h_bytes_per_step=blk_bytes / max(its, 1), seconds=t_e2e, iterations=its,
               call="block_cg_solve_host_ex, zero initial guess (B host->device, solve to tol, X device->host)",
               launches=cm.launch_count() - l1)

    # ---- CPU oracle on a bounded sample, same run ----------------------------------------------------------------
    if not args.no_cpu_baseline:
        from oracle import oracle
        Xfull = cm.fill_block(dims, nb, s, tdt, seed, synth.TAG_X).cpu().numpy().astype(np.complex128)
        Ks = np.eye(s, dtype=np.complex128) * 0.5
        oracle_sample_step(dims, nb, s, sites[:64], A_s[:64], Xfull, Ks)       # warm-up
        dts = []
        while sum(dts) < args.cpu_seconds and len(dts) < 50:                    # bounded: about cpu_seconds of CPU work
            dts.append(oracle_sample_step(dims, nb, s, sites, A_s, Xfull, Ks))
        dt = float(sum(dts))
        cpu = dict(value=len(dts) * step_flops(len(sites), nb, s) / dt / 1e12, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                   sample=f"{len(dts)} steps on {len(sites)} of {V} sites (operator bits read back from the device), {dt:.1f} s in total")

    # ---- SURVEY.md 8(f) NEXT rows on the same operator (never fatal: a failure is recorded in the line) ----------------------
    next_rows = None
    if args.next_rows and dtype == "c64":
        try:
            next_rows = next_rows_point(torch, cm, op, dims, nb, s, c, B, peaks)
        except Exception as e:                                               # noqa: BLE001
            next_rows = dict(error=f"{type(e).__name__}: {e}")
            print(f"bench.py: WARNING next_rows failed: {next_rows['error']}", file=sys.stderr)

    # ---- the other BASELINE.json configurations (parity cases; one time-boxed apply + solve each) --------------------------
    op.close()
    del B, X, Xs
    torch.cuda.empty_cache()
    per_config = []
    if args.per_config:
        for idx in (0, 1, 2, 4):
            if idx != args.config:
                per_config.append(per_config_point(torch, cm, idx, peaks))

    if dtype == "c128":
        dtype_label = "f64"
    elif kernel_name.startswith("stencil_h16"):
        dtype_label = "f32 (fp16x3 split multiply on tcgen05, f32 accumulate)"
    elif kernel_name.startswith("stencil_tc"):
        dtype_label = "f32 (tf32x3 split multiply on tcgen05, f32 accumulate)"
    else:
        dtype_label = "f32"
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=W, ms_per_step=ms / K,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype=dtype_label,
                data="synthetic", metric_note=METRIC_NOTE,
                config=dict(workload=cfg["name"], dims=list(dims), nbasis=nb, nrhs=s, storage=dtype, stencil_points=81,
                            operator_bytes=81 * V * nb * nb * esize, parallelism="replicas only" if world > 1 else "1 GPU",
                            l2="inputs (27.5 GB operator) larger than L2; no flush", diagonal_shift_c=c),
                clocks=clk, e2e=e2e, gpu_launches=int(launches), roofline=roofline, cpu_baseline=cpu,
                sweep=sweep, block_cg_solve=bcg, cheby_solve=cheb, per_config=per_config, next_rows=next_rows,
                peaks={k: v for k, v in peaks.items() if k != "source"}, peaks_source=peaks["source"],
                step_breakdown=dict(apply_ms=a_ms, other_ms=ms / K - a_ms, final_recursive_rel_res=max(out["rel_res_recursive"])))
    print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--nrhs", type=int, default=16)
    ap.add_argument("--config", type=int, default=3, help="index into BASELINE.json configs (default 3: the Nrhs-sweep workload)")
    ap.add_argument("--no-sweep", dest="sweep", action="store_false")
    ap.add_argument("--no-per-config", dest="per_config", action="store_false", help="skip the apply + solve of the other BASELINE configurations")
    ap.add_argument("--no-next-rows", dest="next_rows", action="store_false", help="skip the measurements of the SURVEY 8(f) NEXT rows")
    ap.add_argument("--peaks", action="store_true", help="only measure the roofline denominators of this device and print them as JSON")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cheby-order", type=int, default=120, help="order of the Chebyshev coarse solve timed beside block CG (0: skip)")
    ap.add_argument("--cpu-sites", type=int, default=4096, help="sampled sites of the cpu_baseline leg")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="CPU time budget of the cpu_baseline leg")
    ap.add_argument("--ref-sites", type=int, default=384, help="sampled sites per step of --impl reference")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                             # timing rule: at least 3 warm-up steps
    cfg = synth.config(args.config)
    if args.impl == "reference":
        return run_reference(args, cfg)
    if args.peaks:
        import torch
        import paper_2409_03904_b200 as cm
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
        clocks = ClockSampler(int(os.environ.get("LOCAL_RANK", "0")))
        clocks.start()
        pk = live_peaks(cm, measured_peaks())
        for _ in range(3):                         # a second's worth of samples for the clock record
            cm.measure_peaks()
        pk["clocks"] = clocks.stop()
        print(json.dumps(pk))
        return 0
    return run_ours(args, cfg)


if __name__ == "__main__":
    sys.exit(main())
