#!/usr/bin/env python
"""bench.py - the driver's measurement contract for the B200-native Wilson-Dirac / Neuberger-Dirac hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference]

ONE step = one pass of the whole hot path over one source field on the
BASELINE.json headline lattice 32^3x64 (config index 2: Haar-random SU(3) links, Gaussian source, m = -1.6):
one application of the Neuberger-Dirac operator  D_N eta = c (eta + gamma5 sign(Q) eta)  (eq. 2.4 + 2.11) =
2n+1 Wilson-Dirac stencil launches (a2 link reconstruction, a3 Q, a4 Q^2, a5 fused Clenshaw epilogue, a6 sign
assembly), the low-mode projection (a7 block dot / block axpy, a9 BLAS-1 reductions) and the D_N epilogue (a8).
The layout step a1 (pack / unpack) is inside the `e2e` leg, which runs the same step from pinned HOST buffers.

metric  = Wilson-Dirac GFLOP/s at the conventional 1320 flop per site per stencil application (BASELINE.json),
          value = 1320 * V * (2n+1) * steps * n_gpus / time; D_N applications per second are reported alongside.
roofline = the dominant kernel (the Q stencil), timed alone with CUDA events on the launching stream in the same
          run, against the measured HBM copy peak of MEASURED_PEAKS.json (fp32 and fp64; the JSON's `roofline` is the
          line's dtype, `q_kernel` holds every variant).
cpu_baseline / --impl reference = the CPU oracle (oracle/, plain C + numpy, as it stands) on the host cores on a
          bounded sample of the same recipe.

Multi-GPU: the path is single-GPU in the paper ("no communication necessary");
`--gpus N` under torchrun runs N independent replicas (one lattice per GPU, different sources), no data-path
collective, scaling = weak.  Timing: barrier + synchronize, CUDA events, max over ranks.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_SITE = 1320           # BASELINE.json metric convention
METRIC = "Wilson-Dirac GFLOP/s (1320 flop/site)"
M_KERNEL = -1.6                # kernel mass m = -rho (BASELINE.json configs 2-5)
RHO = 1.6


# ------------------------------------------------------------------------------------------------ helpers
def q_bytes_per_site(prec, recon, n_extra_vectors=0):
    """Algorithmic (compulsory) bytes per site of one stencil launch:
    input spinor once + output once + the site's 4 links once (+ the epilogue's extra vector reads)."""
    return (24 + 24 + 4 * recon + 24 * n_extra_vectors) * (prec // 8)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_traffic(kernel_key):
    """DRAM bytes per launch of the dominant kernel from the committed ncu --set full summary, or None."""
    p = os.path.join(ROOT, "profiles", "q_kernel_dram_traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            parts = [s.strip() for s in line.split(",")]
            if len(parts) >= 2 and parts[0] == kernel_key:
                try:
                    return float(parts[1])
                except ValueError:
                    return None
    return None


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons every 200 ms while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [s.strip() for s in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
                power.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def max_over_ranks(ms, world, backend_device=None):
    """The contract's timing rule: the job's time is the slowest rank's.  Works with NCCL (cuda tensor) and gloo
    (cpu tensor; used by tests/test_bench_host.py at world_size 2)."""
    if world == 1:
        return float(ms)
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(ms)], dtype=torch.float64, device=backend_device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank, world, ms):
    """value = the units ALL ranks processed / the max-over-ranks time (weak scaling, replicas)."""
    return units_per_rank * world / (ms * 1e-3)


# --------------------------------------------------------------------------------------------- CUDA arm
def build_modes(ctx, l, seed=99):
    """l orthonormal vectors and their Rayleigh quotients nu_k = <v_k, Q v_k> for the projection leg (every call
    goes through the C ABI: nd_gaussian, nd_block_dot, nd_block_axpy, nd_scale, nd_apply_Q, nd_dot)."""
    if l == 0:
        return None, np.zeros(0)
    V = ctx.new_spinor(l)
    for k in range(l):
        ctx.gaussian(V[k], seed + k)
        for _ in range(2):
            if k > 0:
                c = ctx.block_dot(V[:k], V[k])
                ctx.block_axpy(-c, V[:k], V[k])
        ctx.scale(1.0 / np.sqrt(ctx.norm2(V[k])), V[k])
    nu = np.zeros(l)
    t = ctx.new_spinor()
    for k in range(l):
        ctx.apply_Q(t, V[k], M_KERNEL)
        nu[k] = ctx.dot(V[k], t).real
    return V, nu


def time_region(torch, ctx, fn, reps):
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    ctx.synchronize()
    e0.record(ctx.stream)
    for _ in range(reps):
        fn()
    e1.record(ctx.stream)
    ctx.synchronize()
    return e0.elapsed_time(e1)


def measure_q_kernel(torch, nd, dims, U64, prec, recon, peak, reps=40, warm=5):
    """The Q stencil alone: fixed source, separate destination, CUDA events on the launch stream."""
    ctx = nd.Context(dims, prec=prec, recon=recon, bc_time=-1)
    ctx.set_gauge(U64.astype(np.complex64) if prec == 32 else U64)
    x, y = ctx.new_spinor(), ctx.new_spinor()
    ctx.gaussian(x, 5636)
    f = lambda: ctx.apply_Q(y, x, M_KERNEL)
    for _ in range(warm):
        f()
    ms = time_region(torch, ctx, f, reps) / reps
    V = ctx.V
    gbs = q_bytes_per_site(prec, recon) * V / (ms * 1e-3) / 1e9
    out = {"prec": prec, "recon": recon, "us_per_launch": ms * 1e3, "gflops_1320": FLOP_PER_SITE * V / (ms * 1e-3) / 1e9,
           "bytes_per_site": q_bytes_per_site(prec, recon), "achieved_gbs": gbs, "frac_of_measured_peak": gbs / peak,
           "frac_of_8TBs": gbs / 8000.0}
    ctx.close()
    del x, y
    torch.cuda.empty_cache()
    return out


def cpu_baseline_sample(steps=1, n=40, l=4, dims=(32, 16, 16, 16)):
    """The oracle as it stands on the host cores: its D_N recipe (oracle/sign.py eq. 2.11 + 2.4 over the plain-C
    stencil oracle/wilson_ref.c) on a bounded sample: a 16^3x32 lattice of the same field recipe, degree n (about 10 s of CPU work per step)."""
    from lattice_inputs import gauge_field, gaussian_spinor
    from oracle import lowmodes as olow
    from oracle import sign as osign
    from oracle import wilson, wilson_c

    U = gauge_field(dims, "haar")
    eta = gaussian_spinor(dims)
    Q = wilson_c.make_Q(U, M_KERNEL, -1)
    qnorm = wilson.norm_bound_Q(M_KERNEL)
    eps = 0.002
    c = osign.cheb_coeffs(n, eps)
    rng = np.random.Generator(np.random.PCG64(3))
    Vs = olow.orthonormalise([rng.standard_normal(eta.shape) + 1j * rng.standard_normal(eta.shape) for _ in range(l)])
    nu, Us = osign.rayleigh_ritz_Q(Q, Vs)
    osign.apply_DN(Q, wilson.apply_gamma5, eta, c[:3], eps, qnorm, 1.0 / RHO, nu, Us)    # warm-up (loads the C library)
    t0 = time.perf_counter()
    for _ in range(steps):
        osign.apply_DN(Q, wilson.apply_gamma5, eta, c, eps, qnorm, 1.0 / RHO, nu, Us)
    dt = (time.perf_counter() - t0) / steps
    vol = int(np.prod(dims))
    gflops = FLOP_PER_SITE * vol * (2 * n + 1) / dt / 1e9
    return {"value": gflops, "unit": "GFLOP/s", "cores": wilson_c.num_threads(), "kind": "oracle",
            "sample": f"oracle D_N recipe (oracle/sign.py over oracle/wilson_ref.c, fp64, full 3x3 links) on a "
                      f"{dims[1]}^3x{dims[0]} Haar lattice, degree n={n}, l={l}: {2 * n + 1} stencils/step, "
                      f"{dt:.2f} s/step",
            "dn_applies_per_s": 1.0 / dt, "seconds_per_step": dt}


def run_b200(args):
    import torch

    import paper_1010_5636_b200 as nd
    from lattice_inputs import gauge_field, parse_lattice

    rank, world, local = dist_env()
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("--gpus N > 1 must be launched with torch.distributed.run (one rank per GPU)")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the CUDA path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dims = parse_lattice(args.lattice)
    prec, recon, n, l = args.prec, args.recon, args.degree, args.lowmodes
    peak, peak_src = load_peaks()

    # BASELINE config 2: Haar-random links, seeded (configs 1, 3, 4: --field smooth)
    U64 = gauge_field(dims, args.field, eps=args.field_eps)
    ctx = nd.Context(dims, prec=prec, recon=recon, bc_time=-1, device=local)
    ctx.set_gauge(U64.astype(np.complex64) if prec == 32 else U64)
    V = ctx.V
    qnorm = abs(4.0 + M_KERNEL) + 4.0
    c, delta = nd.cheb_coeffs(n, args.eps)
    ctx.set_sign_poly(c, args.eps, qnorm, M_KERNEL)
    eig = None
    if args.eigensolve and l > 0:
        # BASELINE config 4: the low modes come from the library's own eigen-solver (a10), timed on the host clock
        # (it synchronises for its small dense problems); eps then follows DESIGN.md R11.
        ctx.synchronize()
        t0 = time.perf_counter()
        modes, nu, resid, st = ctx.lowmodes_compute(max(1, l - l // 8), M_KERNEL, tol=args.eig_tol, maxit=60, lextra=max(8, l // 4),
                                                    degree=args.eig_degree, l_max=l + l // 8, stop="bound")
        l = st["l_chosen"]
        ctx.synchronize()
        eig = {"seconds": time.perf_counter() - t0, "l": l, "tol_bound_2_10": args.eig_tol, "converged": st["converged"],
               "outer_iterations": st["iterations"], "q_stencils": st["stencils"], "max_residue_Q": float(resid.max()),
               "nu2_min": float((nu ** 2).min()), "nu2_max": float((nu ** 2).max())}
        eig["l_chosen"] = l
        eig["kappa_pm"] = [float(st["kappa"][0]), float(st["kappa"][1])]                 # eq. 2.9
        eig["projector_bound_pm"] = [float(b) if np.isfinite(b) else None for b in st["bound"]]   # eq. 2.10
        args.eps = 0.99 * float((nu ** 2).max()) / qnorm ** 2
        c, delta = nd.cheb_coeffs(n, args.eps)
        ctx.set_sign_poly(c, args.eps, qnorm, M_KERNEL)
    else:
        modes, nu = build_modes(ctx, l)
    ctx.set_lowmodes(modes, nu)
    eta, out, work = ctx.new_spinor(), ctx.new_spinor(), ctx.new_spinor(3)
    ctx.gaussian(eta, 5636 + rank)                        # replicas: a different source per rank
    step = lambda: ctx.apply_DN(out, eta, 1.0 / RHO, work, use_graph=True)

    # ---- device-resident leg
    for _ in range(args.warmup):
        step()
    ctx.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = ctx.launch_count()
    ms = time_region(torch, ctx, step, args.steps)
    launches = ctx.launch_count() - l0
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = max_over_ranks(ms, world, torch.device("cuda", local))
    clocks = sampler.stop() if rank == 0 else None
    stencils = 2 * n + 1
    gflop_per_step = FLOP_PER_SITE * V * stencils / 1e9
    value = whole_job_value(gflop_per_step * args.steps, world, ms)

    # ---- end-to-end leg: host AoS source in pinned memory -> pack -> D_N -> unpack -> pinned host result
    cdt = torch.complex64 if prec == 32 else torch.complex128
    h_in = torch.empty(dims + (4, 3), dtype=cdt, pin_memory=True)
    h_out = torch.empty(dims + (4, 3), dtype=cdt, pin_memory=True)
    h_in.copy_(torch.view_as_complex(torch.randn(dims + (4, 3, 2), dtype=torch.float32 if prec == 32 else torch.float64)))

    def e2e_step():
        ctx.pack_spinor_host(h_in.data_ptr(), prec, eta)
        ctx.apply_DN(out, eta, 1.0 / RHO, work, use_graph=True)
        ctx.unpack_spinor_host(out, h_out.data_ptr(), prec)      # synchronises (host result)

    for _ in range(2):
        e2e_step()
    if world > 1:
        dist.barrier()
    ms_e2e = time_region(torch, ctx, e2e_step, args.steps)
    ms_e2e = max_over_ranks(ms_e2e, world, torch.device("cuda", local))
    e2e_value = whole_job_value(gflop_per_step * args.steps, world, ms_e2e)
    hbytes = V * 24 * (prec // 8)

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return
    # ---- rank 0 only: the dominant kernel alone (roofline), every variant; the CPU oracle
    ctx.close()
    del modes, eta, out, work
    torch.cuda.empty_cache()
    qk = {}
    for p, r in ((32, 12), (64, 12), (32, 8), (64, 8), (32, 18), (64, 18)):
        if args.quick and (p, r) not in ((prec, recon),):
            continue
        qk[f"f{p}_recon{r}"] = measure_q_kernel(torch, nd, dims, U64, p, r, peak)
    main = qk[f"f{prec}_recon{recon}"]
    roofline = {"bound": "hbm", "achieved": main["achieved_gbs"], "peak": peak, "unit": "GB/s",
                "frac": main["achieved_gbs"] / peak, "traffic": load_traffic(f"f{prec}_recon{recon}"),
                "kernel": "wilson_Q_kernel (Q stencil, plain epilogue)", "peak_source": peak_src,
                "algorithmic_bytes_per_launch": main["bytes_per_site"] * V, "us_per_launch": main["us_per_launch"],
                "frac_of_8TBs_nominal": main["achieved_gbs"] / 8000.0}
    cpu = None if args.no_cpu_baseline else cpu_baseline_sample()
    line = {
        "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if prec == 32 else "f64", "data": "synthetic",
        "config": {"workload": f"D_N apply (eq. 2.4+2.11) on {args.lattice}, {args.field} SU(3) links, m=-1.6, recon {recon}, "
                               f"degree n={n} (2n+1={stencils} Q stencils), l={l} projected modes, CUDA graph",
                   "lattice": args.lattice, "sites": V, "recon": recon, "degree": n, "eps": args.eps, "delta": delta,
                   "lowmodes": l, "replicas": world, "parallelism": f"replicas x{world}",
                   "l2_policy": "inputs larger than L2 (links + vectors >= 1.4 GB fp32), no flush needed"},
        "dn_applies_per_s": world * args.steps / (ms * 1e-3),
        "q_stencils_per_s": world * args.steps * stencils / (ms * 1e-3),
        "e2e": {"value": e2e_value, "unit": "GFLOP/s", "h2d_bytes_per_step": hbytes, "d2h_bytes_per_step": hbytes,
                "ms_per_step": ms_e2e / args.steps},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": roofline,
        "q_kernel": qk,
        "cpu_baseline": cpu,
    }
    if eig is not None:
        line["eigensolve"] = eig
    print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------- reference arm
def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return
    # W warm-up + K timed steps of the oracle, each step one D_N application on the bounded sample
    cpu_baseline_sample(steps=max(args.warmup, 1), n=2)
    r = cpu_baseline_sample(steps=args.steps)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": "GFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["seconds_per_step"] * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "CPU oracle: " + r["sample"]},
        "cpu_baseline": {"value": r["value"], "unit": "GFLOP/s", "kind": "oracle", "cores": r["cores"], "sample": r["sample"]},
        "e2e": {"value": r["value"], "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--lattice", default="32^3x64")
    ap.add_argument("--prec", type=int, default=32, choices=[32, 64])
    ap.add_argument("--recon", type=int, default=12, choices=[18, 12, 8])
    ap.add_argument("--degree", type=int, default=100)
    ap.add_argument("--eps", type=float, default=0.002)
    ap.add_argument("--lowmodes", type=int, default=8)
    ap.add_argument("--field", default="haar", choices=["haar", "smooth"], help="gauge field recipe (DESIGN.md section 4)")
    ap.add_argument("--field-eps", type=float, default=0.25, help="eps of U = exp(i eps H) for --field smooth")
    ap.add_argument("--eigensolve", action="store_true", help="low modes from nd_lowmodes_compute (timed), eps by R11")
    ap.add_argument("--eig-tol", type=float, default=1e-2, help="stop when the bound (2.10) on the projector error is below this")
    ap.add_argument("--eig-degree", type=int, default=80)
    ap.add_argument("--quick", action="store_true", help="time only the line's own Q-kernel variant")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
