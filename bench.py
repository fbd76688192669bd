#!/usr/bin/env python
"""bench.py -- throughput of the nonlinear E×B hot path (gx_nonlinear_rhs) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cyclone] [--impl reference]

One "step" = one gx_nonlinear_rhs call (all rows a1-a8 of DESIGN.md) on one batch of seeded synthetic
input of the named configuration.  Prints ONE JSON line (rank 0).  Timing: CUDA events on the launch
stream, bracketed by barrier + synchronize, max over ranks.  The inputs rotate through buffer sets
whose total size exceeds the 126 MB L2 so that g is read from and out written to HBM every step.

--impl reference times the fp64 CPU oracle (oracle/gx_oracle.py, as it stands) on a bounded sample
of the same workload on the host cores; it is a deliberately slow baseline, not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2209_06731_b200 import dist as D          # noqa: E402
from paper_2209_06731_b200 import inputs as I        # noqa: E402

METRIC = "nonlinear_rhs_evals_per_s"
UNIT = "evals/s"
FP32_LANES_PER_SM = 128
L2_BYTES = 126e6


def workload_name(cfg):
    return (f"{cfg.name}: Nx={cfg.Nx} Ny={cfg.Ny} Nz={cfg.Nz} Nl={cfg.Nl} Nm={cfg.Nm} Ns={cfg.Ns} "
            f"(nakx={cfg.nakx} naky={cfg.naky} J={cfg.nj})")


# ------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons with NVML in a thread while the timed region runs.  The thread starts
    sampling when arm() is called -- by the timed loop right after its last launch is enqueued, while the GPU still
    works through the queue -- so that no NVML call competes with the kernel launches for the driver."""

    def __init__(self, index=0, period=0.01):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.period, self._stop, self._thr, self.ok = period, threading.Event(), None, False
        self._armed = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            pynvml.nvmlDeviceGetClockInfo(self.h, pynvml.NVML_CLOCK_SM)           # first-use cost of the queries, discarded
            pynvml.nvmlDeviceGetCurrentClocksEventReasons(self.h)
            self.ok = True
        except Exception:
            self.ok = False

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80, "sw_power_cap": 0x4}
        self._armed.wait()
        while True:
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            if self._stop.wait(self.period):
                break

    def __enter__(self):
        if self.ok and self._thr is None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def arm(self):
        self._armed.set()

    def __exit__(self, *a):
        self._stop.set()
        self._armed.set()
        if self._thr:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------- CPU oracle leg
def oracle_sample(cfg, geo, budget_s=12.0):
    """Times oracle.nonlinear_rhs (pseudo-spectral naive-DFT path, fp64, as it stands) on a bounded sample
    of the workload: whole evaluations when one fits the budget, else a subset of the independent
    (s,m,z) planes scaled to a whole evaluation.  -> (evals/s, description, seconds spent)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import gx_oracle as O
    sm_all = [(s, m) for s in range(cfg.Ns) for m in range(cfg.Nm)]
    small = int(np.prod(cfg.g_shape)) <= 4_500_000
    sm_sel = sm_all if small else sm_all[:: max(1, len(sm_all) // 4)][:4]
    need_sm = sorted(set(sm_sel) | {(s, 0) for s in range(cfg.Ns)})
    G = I.make_state(cfg, geo, planes=None if small else need_sm)
    Phi = O.field_solve(G, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, tau_fac=cfg.tau_fac,
                        adiabatic=(cfg.Ns == 1)).astype(np.complex64)
    n_all = len(sm_all) * cfg.Nz
    cand = [(s, m, z) for (s, m) in sm_sel for z in range(cfg.Nz)]

    def run(planes):
        return O.nonlinear_rhs(G, Phi, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species,
                               method="dft", planes=planes)

    probe = cand[:: max(1, len(cand) // 4)][:4]
    t0 = time.perf_counter()
    run(probe)
    per_plane = (time.perf_counter() - t0) / len(probe)
    if small and per_plane * n_all <= budget_s:
        n = max(1, int(budget_s / (per_plane * n_all)))
        t0 = time.perf_counter()
        for _ in range(n):
            run(None)
        dt = time.perf_counter() - t0
        return n / dt, f"{n} whole evaluations ({n_all} (s,m,z) planes each); oracle path B (naive DFT, fp64)", dt
    k = max(len(probe), min(len(cand), int(budget_s / per_plane)))
    planes = cand[:: max(1, len(cand) // k)][:k]
    t0 = time.perf_counter()
    run(planes)
    dt = time.perf_counter() - t0
    return ((len(planes) / n_all) / dt,
            f"{len(planes)} of {n_all} independent (s,m,z) planes, scaled to a whole evaluation; "
            f"oracle path B (naive DFT, fp64)", dt)


def host_threads():
    try:
        from threadpoolctl import threadpool_info
        n = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
        return int(n)
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank, _, world = D.env_world()
    if rank != 0:
        return 0
    cfg = I.named_config(args.config)
    geo = I.geometry_arrays(cfg)
    # every step is a bounded sample of the workload; the per-step budget shrinks with --steps so that the whole
    # run (warm-up included) stays within about two minutes
    steps, warm = max(1, args.steps), max(0, args.warmup)
    budget = max(0.25, min(10.0, 90.0 / (steps + warm)))
    for _ in range(warm):
        oracle_sample(cfg, geo, budget_s=budget)
    vals, secs, sample = [], 0.0, ""
    for _ in range(steps):
        v, sample, dt = oracle_sample(cfg, geo, budget_s=budget)
        vals.append(v)
        secs += dt
    value = float(np.mean(vals))
    cores = host_threads()
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": warm, "ms_per_step": 1e3 / value, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "note": "fp64 CPU oracle on host cores; bounded sample per step"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------- library reference point
def cufft_composition(torch, cfg, grid, g, phi, ours, steps=20):
    """The paper's own design for this step (batched cuFFT + cuBLAS for the Laguerre
    matrices + pointwise kernels), composed from torch.fft (cuFFT) and torch.einsum (cuBLAS) on the same
    tables and inputs.  A reference point on the same GPU, not part of the product path.
    -> (evals/s, max-norm relative difference to `ours`)."""
    from paper_2209_06731_b200 import binding as B
    dev = g.device
    Ns, Nm, Nl, Nz, nakx, naky = cfg.g_shape
    nj, Nx, Ny = cfg.nj, cfg.Nx, cfg.Ny
    T, Tinv, M = B.gx_export_tables(grid.h, Nl, Ns * Nz * nj * nakx * naky)
    Tt = torch.from_numpy(T).to(dev).to(torch.complex64)
    Ti = torch.from_numpy(Tinv).to(dev).to(torch.complex64)
    Mt = torch.from_numpy(M.reshape(Ns, Nz, nj, nakx, naky)).to(dev)
    K = (nakx - 1) // 2
    kxi = torch.tensor([i if i <= K else i - nakx for i in range(nakx)], device=dev)
    rows = torch.where(kxi >= 0, kxi, kxi + Nx)
    ikx = (1j * cfg.dkx * kxi.to(torch.float32)).to(torch.complex64)[:, None]
    iky = (1j * cfg.dky * torch.arange(naky, device=dev, dtype=torch.float32)).to(torch.complex64)[None, :]
    Nyc = Ny // 2 + 1

    def to_real(f):
        pad = torch.zeros(f.shape[:-2] + (Nx, Nyc), dtype=torch.complex64, device=dev)
        pad[..., rows, :naky] = f
        return torch.fft.irfft2(pad, s=(Nx, Ny), norm="forward")

    def step():
        chi = Mt * phi[None, :, None]                                    # [s][z][j][kx][ky]
        gt = torch.einsum("jl,smlzxy->smzjxy", Tt, g)
        dxc, dyc = to_real(ikx * chi)[:, None], to_real(iky * chi)[:, None]
        br = dyc * to_real(ikx * gt) - dxc * to_real(iky * gt)
        bh = torch.fft.rfft2(br, norm="forward")[..., rows, :naky]
        return -torch.einsum("lj,smzjxy->smlzxy", Ti, bh)

    out = step()
    err = float((out - ours).abs().max() / ours.abs().max())
    for _ in range(2):
        step()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    return steps / (e0.elapsed_time(e1) * 1e-3), err


# ------------------------------------------------------------------------------- measured FP32 peak
def fp32_ubench(B, sm_mhz, n_sm, full=False):
    """FP32 pipe micro-benchmark of the library (gx_ubench_fp32): lane operations per clock and SM for the scalar
    and packed add / mul / fma, at 2 x 512 threads per SM (and more shapes with --ubench)."""
    out = {}
    shapes = [(512, 2)] + ([(256, 2), (192, 2), (1024, 1), (384, 1)] if full else [])
    for kind, name in enumerate(B.UBENCH_KINDS):
        for nt, bps in shapes:
            best = 0.0
            try:
                for _ in range(3):
                    ms, ops = B.gx_ubench_fp32(kind, nt, bps, 4096)
                    best = max(best, ops / (ms * 1e-3))
            except B.GxError:
                continue                                  # launch shape not possible for this kernel (registers)
            key = name if (nt, bps) == (512, 2) else f"{name} @{bps}x{nt}"
            out[key] = {"lane_ops_per_s": best, "lane_ops_per_clk_per_sm": best / (sm_mhz * 1e6) / n_sm}
    return out


# ------------------------------------------------------------------------------- tensor-core DFT question
def run_tcdft(args):
    """`--tcdft`: would the radix-16 stages pay as split-TF32 matrix products on the tensor cores?  Measures
    (i) the library's register radix-16 (scalar and packed), (ii) the TF32 and BF16 tensor rates of this GPU on a
    large library GEMM (cuBLAS, which runs tcgen05 kernels on sm_100a: an upper bound for any hand-written tile),
    (iii) the accuracy of the 3-term split DFT16 = Xh Wh + Xh Wl + Xl Wh on the tensor cores against fp64.  A
    16-point complex DFT as a real matrix product is a [32 x 32] matrix per vector: 1024 MACs, x3 for the split."""
    import torch
    from paper_2209_06731_b200 import binding as B
    dev = torch.device("cuda", 0)
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    clk = (peaks.get("sm_max_mhz") or 1965.0) * 1e6
    out = {"leg": "tcdft", "n_sm": n_sm, "sm_clock_mhz": clk / 1e6}
    # (i) register radix-16
    for packed, name in [(0, "radix16_scalar"), (1, "radix16_packed")]:
        best = 0.0
        for nt, bps in [(192, 2), (256, 2), (128, 4)]:
            try:
                ms, n = B.gx_ubench_dft16(packed, nt, bps, 512)
                best = max(best, n / (ms * 1e-3))
            except B.GxError:
                pass
        out[name] = {"transforms_per_s": best, "cycles_per_transform_per_sm": clk * n_sm / best}
    # (ii) tensor rates on a large GEMM
    def gemm_rate(dtype, allow_tf32):
        torch.backends.cuda.matmul.allow_tf32 = allow_tf32
        n = 8192
        a = torch.randn(n, n, device=dev, dtype=dtype)
        b = torch.randn(n, n, device=dev, dtype=dtype)
        for _ in range(2):
            a @ b
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(5):
            a @ b
        e1.record()
        torch.cuda.synchronize()
        return 5 * 2.0 * n ** 3 / (e0.elapsed_time(e1) * 1e-3)
    tf32 = gemm_rate(torch.float32, True)
    bf16 = gemm_rate(torch.bfloat16, False)
    fp32 = gemm_rate(torch.float32, False)
    out["gemm_flops_per_s"] = {"tf32": tf32, "bf16": bf16, "fp32_cuda_cores": fp32}
    macs = 32 * 32
    for name, rate, terms in [("dft16_as_tf32_3term", tf32, 3), ("dft16_as_bf16_6term", bf16, 6)]:
        cyc = terms * 2.0 * macs / (rate / (clk * n_sm))
        out[name] = {"cycles_per_transform_per_sm_upper_bound": cyc,
                     "note": "tensor pipe only at the measured library GEMM rate: no operand split, staging or TMEM read-back"}
    # (iii) accuracy of the 3-term split on the real tensor cores
    torch.backends.cuda.matmul.allow_tf32 = True
    nb = 1 << 16
    x = torch.randn(nb, 32, device=dev, dtype=torch.float64)
    k = torch.arange(16, device=dev, dtype=torch.float64)
    ang = 2.0 * np.pi * torch.outer(k, k) / 16.0
    c, sn = torch.cos(ang), torch.sin(ang)
    w = torch.zeros(32, 32, device=dev, dtype=torch.float64)      # interleaved (re, im): y = x W, inverse DFT e^{+i ang}
    w[0::2, 0::2], w[0::2, 1::2], w[1::2, 0::2], w[1::2, 1::2] = c, sn, -sn, c
    ref = x @ w
    def tf32_round(t):                                          # keep 10 explicit mantissa bits (round to nearest even)
        i = t.float().view(torch.int32)
        i = (i + 0x00000FFF + ((i >> 13) & 1)) & ~0x1FFF
        return i.view(torch.float32)
    xf, wf = x.float(), w.float()
    xh, wh = tf32_round(xf), tf32_round(wf)
    xl, wl = xf - xh, wf - wh
    y1 = (xh @ wh).double()
    y3 = ((xh @ wh) + (xh @ wl) + (xl @ wh)).double()
    scale = ref.abs().max()
    torch.backends.cuda.matmul.allow_tf32 = False
    yf = (xf @ wf).double()
    out["accuracy_vs_fp64"] = {"tf32_1term": float((y1 - ref).abs().max() / scale), "tf32_3term": float((y3 - ref).abs().max() / scale),
                               "fp32_matmul": float((yf - ref).abs().max() / scale)}
    out["split_cost_lane_ops_per_transform"] = 2 * 32      # per real: one rounding op and one subtraction on the CUDA cores
    r = out["radix16_packed"]["cycles_per_transform_per_sm"]
    out["verdict"] = ("tensor form needs %.2f cycles per transform and SM at best (TF32, 3 terms) + %.2f cycles of FP32 pipe for the operand "
                      "split, against %.2f measured for the register radix-16: not adopted" %
                      (out["dft16_as_tf32_3term"]["cycles_per_transform_per_sm_upper_bound"], 64 / 123.0, r))
    print(json.dumps(out))
    return 0


# ------------------------------------------------------------------------------- GPU leg
def run_gpu(args):
    import torch
    from paper_2209_06731_b200 import binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    rank, local_rank, world = D.init("nccl") if int(os.environ.get("WORLD_SIZE", "1")) > 1 else (0, 0, 1)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    cfg = I.named_config(args.config)
    geo = I.geometry_arrays(cfg)
    # weak scaling: ONE seeded state with Nm*world Hermite moments, rank r owns the block [m0, m1) (the paper's
    # own decomposition); phi is replicated: every rank solves quasineutrality from the m = 0 slab
    m0, m1, Nm_global = D.hermite_block(cfg.Nm, rank, world)
    cfg_global = I.Config(**{**cfg.__dict__, "Nm": Nm_global})
    grid = B.Grid(cfg, geo)
    flops = grid.query(B.GX_Q_NL_FLOPS)
    alg_bytes = grid.query(B.GX_Q_NL_BYTES)
    launches_per_call = grid.query(B.GX_Q_LAUNCHES_PER_NL)

    # this rank's Hermite block of the global seeded state; phi from the library's own field solve (product path)
    # on the global m = 0 slab (a one-moment handle: the field solve reads m = 0 only)
    g_elems = int(np.prod(cfg.g_shape))
    set_bytes = 2 * g_elems * 8 + int(np.prod(cfg.phi_shape)) * 8
    nsets = max(2, int(np.ceil(4.2 * L2_BYTES / set_bytes)))
    nsets = min(nsets, max(2, int(40e9 // set_bytes)))
    G0 = I.make_state(cfg_global, geo, hermite_block=(m0, m1))
    g_host = torch.from_numpy(G0)
    cfg_m0 = I.Config(**{**cfg.__dict__, "Nm": 1})
    grid_m0 = B.Grid(cfg_m0, geo)
    g_m0 = torch.from_numpy(I.make_state(cfg_global, geo, hermite_block=(0, 1))).to(dev)
    gs, phis, outs = [], [], []
    for k in range(nsets):
        g = g_host.to(dev)
        scale_k = 1.0 + 0.01 * k            # distinct contents per set, same spectrum
        if k:
            g.mul_(scale_k)
        phi = torch.empty(cfg.phi_shape, dtype=torch.complex64, device=dev)
        grid_m0.field_solve(g_m0, phi)
        phi.mul_(scale_k)                   # the field solve is linear in g
        gs.append(g); phis.append(phi); outs.append(torch.empty_like(g))
    torch.cuda.synchronize()
    grid_m0.close()

    def step(i):
        k = i % nsets
        grid.nonlinear_rhs(gs[k], phis[k], outs[k])

    sampler = ClockSampler(local_rank)      # NVML initialised and the (idle) thread started before the warm-up, not at
    sampler.__enter__()                     # the edge of the timed region
    for i in range(args.warmup):
        step(i)
    torch.cuda.synchronize()
    D.barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with sampler as clk:
        torch.cuda.synchronize()
        ev0.record()
        for i in range(args.steps):
            step(i)
        ev1.record()
        clk.arm()                           # everything is enqueued: sample the clocks while the GPU runs it
        torch.cuda.synchronize()
    D.barrier()
    sec = ev0.elapsed_time(ev1) * 1e-3
    value, sec_max = D.aggregate_throughput(float(args.steps), sec, device=dev)
    assert all(torch.isfinite(o.real).all() for o in outs[:2])

    # per-kernel durations, live, same launch configuration (events around each kernel)
    B.gx_profile_set(grid.h, 1)
    nprof = min(args.steps, 200)
    for i in range(nprof):
        step(i)
    kms, ncalls = B.gx_profile_get(grid.h)
    B.gx_profile_set(grid.h, 0)
    kern_us = [1e3 * t / max(ncalls, 1) for t in kms]

    # end-to-end through the host entry point: pinned host buffers, H2D + compute + D2H every step
    gh = g_host.pin_memory()
    ph = phis[0].cpu().pin_memory()
    oh = torch.empty_like(gh).pin_memory()
    e2e_steps = max(3, min(args.steps, 30))
    for _ in range(3):
        grid.nonlinear_rhs_host(gh, ph, oh)
    torch.cuda.synchronize()
    D.barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        grid.nonlinear_rhs_host(gh, ph, oh)          # synchronises before returning
    torch.cuda.synchronize()
    e2e_sec = time.perf_counter() - t0
    e2e_value, _ = D.aggregate_throughput(float(e2e_steps), e2e_sec, device=dev)

    # the mandated full right-hand side and the SSP-RK3 step, same inputs
    def timed(fn, n):
        for _ in range(3):
            fn(0)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record()
        for i in range(n):
            fn(i)
        b.record()
        torch.cuda.synchronize()
        return n / (a.elapsed_time(b) * 1e-3)

    n_aux = max(3, min(args.steps, 200))
    rhs_rate = timed(lambda i: grid.rhs(gs[i % nsets], outs[i % nsets]), n_aux)
    rhs_linked_rate = None
    try:                                  # same right-hand side with twist-and-shift linked z operators (Eq. 4.29)
        grid_l = B.Grid(cfg, geo, linked=True)
        rhs_linked_rate = timed(lambda i: grid_l.rhs(gs[i % nsets], outs[i % nsets]), n_aux)
        grid_l.close()
    except B.GxError:
        pass
    g_rk = gs[0].clone()
    g_rk.mul_(1e-3)                       # small amplitude; dt from the parallel-streaming CFL (Eq. 5.5)
    vt_max = max(np.sqrt(sp.temp / sp.mass) for sp in cfg.species)
    dt_rk = 0.2 / (vt_max * abs(float(geo["gradpar"])) * (cfg.Nz / 2) * np.sqrt(2.0 * cfg.Nm) + 10.0)
    rk_rate = timed(lambda i: grid.ssprk3_step(g_rk, dt_rk), max(3, n_aux // 3))
    assert torch.isfinite(g_rk.real).all()
    ref_point = None
    if rank == 0 and not args.skip_reference_point and g_elems <= 8_000_000:
        grid.nonlinear_rhs(gs[0], phis[0], outs[0])
        torch.cuda.synchronize()
        try:
            rv, rerr = cufft_composition(torch, cfg, grid, gs[0], phis[0], outs[0])
            ref_point = {"kind": "cuFFT + cuBLAS composition of the same step (torch.fft / torch.einsum), same GPU",
                         "value": rv, "unit": UNIT, "rel_diff_to_ours": rerr}
        except Exception as e:                                  # library leg only; never affects the product numbers
            ref_point = {"kind": "cuFFT + cuBLAS composition", "error": repr(e)[:200]}

    line = None
    if rank == 0:
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        clocks = clk.summary()
        sm_max = peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0
        n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
        peak_tflops = n_sm * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
        # dominant kernel: bracket_kernel.  Its algorithmic flops = whole-call flops minus the chi planes'
        # transforms and multiplies (SURVEY 8d formula with nT = 3P) -- see DESIGN.md "Roofline".
        P = cfg.Ns * cfg.Nm * cfg.Nz * cfg.nj
        SZJ = cfg.Ns * cfg.Nz * cfg.nj
        fft = 5 * cfg.Nx * np.log2(cfg.Nx) * cfg.naky + 2.5 * cfg.Ny * np.log2(cfg.Ny) * cfg.Nx
        nk = cfg.nakx * cfg.naky
        br_flops = 3 * P * fft + 3 * cfg.Nx * cfg.Ny * P + (4 * cfg.nj * cfg.Nl) * nk * cfg.Ns * cfg.Nm * cfg.Nz + 4 * nk * P
        br_sec = kern_us[1] * 1e-6
        br_serial = br_flops / br_sec / 1e12 if br_sec > 0 else 0.0
        # The grids of consecutive calls overlap on the device (row family: the chi planes and the first bracket units of
        # call N+1 run under the tail of call N), so no kernel has a launch duration of its own inside the timed
        # region: the step is the unit.  achieved = algorithmic flops of one call / device time per call of the timed
        # loop (CUDA events, max over ranks); the serialised per-kernel event times are kept beside it.
        step_sec = sec_max / args.steps
        achieved = flops / step_sec / 1e12
        traffic = None
        try:
            traffic = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json"))).get(cfg.name, {}).get("bracket_kernel")
        except Exception:
            pass
        ub = fp32_ubench(B, sm_max, n_sm, full=args.ubench)
        peak_measured = 2.0 * ub["fma.rn.f32"]["lane_ops_per_s"] / 1e12          # FMA = 2 flops per lane operation
        traffic_call = None
        try:
            traffic_call = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json"))).get(cfg.name, {}).get("call")
        except Exception:
            pass
        roofline = {"bound": "alu", "kernel": "chi-planes + bracket grids of one call (%s family; they overlap across calls, the step is the unit)" % B.FAMILY_NAMES.get(grid.query(B.GX_Q_KERNEL_FAMILY), "?"), "achieved": achieved, "peak": peak_tflops,
                    "unit": "TFLOP/s", "frac": achieved / peak_tflops, "traffic": traffic,
                    "peak_measured": peak_measured, "frac_of_measured": achieved / peak_measured,
                    "peak_measured_source": "gx_ubench_fp32: fma.rn.f32, 16 chains per thread, 2 x 512 threads per SM, this run",
                    "fp32_pipe_lane_ops_per_clk_per_sm": {k: round(v["lane_ops_per_clk_per_sm"], 2) for k, v in ub.items()},
                    "traffic_per_call": traffic_call,
                    "peak_source": f"{n_sm} SMs x 128 FP32 lanes x 2 x {sm_max:.0f} MHz (max SM clock, MEASURED_PEAKS.json)",
                    "kernel_us": {"chi_planes": kern_us[0], "bracket": kern_us[1], "laguerre_inverse": kern_us[2]},
                    "kernel_us_note": "each kernel alone (events between the launches serialise them); with a8 inside the bracket kernel the third entry is an empty interval",
                    "bracket_kernel_serialised": {"alg_flops": br_flops, "achieved": br_serial, "frac": br_serial / peak_tflops},
                    "kernel_share_of_step": kern_us[1] / max(sum(kern_us), 1e-9),
                    "whole_call": {"alg_flops": flops, "alg_bytes": alg_bytes,
                                   "frac_of_fp32_peak": flops * value / world / 1e12 / peak_tflops,
                                   "hbm_gbs": alg_bytes * value / world / 1e9,
                                   "hbm_peak_gbs": peaks.get("hbm_gbs")}}
        cpu_v, cpu_sample, _ = (oracle_sample(cfg, geo, budget_s=12.0) if world == 1 and not args.skip_cpu_baseline
                                  else (None, "skipped (N>1 or --skip-cpu-baseline)", 0))
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": 1e3 * sec_max / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": workload_name(cfg), "hermite_moments_global": Nm_global,
                           "parallelism": f"hermite-block x{world} of one seeded state, phi replicated, no collective",
                           "l2": f"inputs rotate through {nsets} buffer sets ({nsets * set_bytes / 1e6:.0f} MB > 126 MB L2)",
                           "grid_point_moments_per_s": value * cfg.grid_point_moments,
                           "phi": "gx_field_solve on device (Boltzmann electrons)" if cfg.Ns == 1 else "gx_field_solve on device"},
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": (g_elems + int(np.prod(cfg.phi_shape))) * 8,
                        "d2h_bytes_per_step": g_elems * 8, "steps": e2e_steps},
                "gpu_launches": launches_per_call * args.steps,
                "kernel_family": B.FAMILY_NAMES.get(grid.query(B.GX_Q_KERNEL_FAMILY), "?"),
                "gx_rhs": {"value": rhs_rate * world, "unit": "full rhs evals/s (field solve + nonlinear + linear)",
                           "twist_shift_linked": None if rhs_linked_rate is None else rhs_linked_rate * world},
                "ssprk3": {"value": rk_rate * world, "unit": "SSP-RK3 steps/s (3 gx_rhs each)"},
                "reference_point": ref_point,
                "roofline": roofline,
                "cpu_baseline": {"value": cpu_v, "unit": UNIT, "cores": host_threads(), "kind": "oracle",
                                 "sample": cpu_sample}}
        print(json.dumps(line))
    grid.close()
    D.finalize()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=100)
    ap.add_argument("--config", default="cyclone", choices=I.CONFIG_NAMES + ["w7x-shape", "nx64", "nx128", "nx192", "nx256"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--skip-cpu-baseline", action="store_true", help="omit the oracle timing (ncu passes)")
    ap.add_argument("--skip-reference-point", action="store_true", help="omit the cuFFT+cuBLAS composition")
    ap.add_argument("--tcdft", action="store_true", help="tensor-core DFT question: radix-16 in registers vs split-TF32 matrix form")
    ap.add_argument("--ubench", action="store_true", help="FP32 pipe micro-benchmark at more launch shapes (roofline.fp32_pipe_...)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    if args.tcdft:
        return run_tcdft(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # no launcher: start one process per GPU ourselves (same command the driver uses)
        import subprocess
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but only {have} CUDA device(s) are visible")
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 2000), os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)
    if int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} does not match WORLD_SIZE={os.environ.get('WORLD_SIZE', '1')}")
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
