#!/usr/bin/env python
"""bench.py - the driver's measurement contract for the B200-native Wilson-Dirac / Neuberger-Dirac hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--quick]

ONE step = one pass of the whole hot path over one source field on the
BASELINE.json headline lattice 32^3x64 (config index 2: Haar-random SU(3) links, Gaussian source, m = -1.6):
one application of the Neuberger-Dirac operator  D_N eta = c (eta + gamma5 sign(Q) eta)  (eq. 2.4 + 2.11) =
2n+1 Wilson-Dirac stencil launches (a2 link reconstruction, a3 Q, a4 Q^2, a5 fused Clenshaw epilogue, a6 sign
assembly), the low-mode projection (a7 block dot / block axpy, a9 BLAS-1 reductions) and the D_N epilogue (a8).
The layout step a1 (pack / unpack) is inside the `e2e` leg, which runs the same step from pinned HOST buffers.

metric   = Wilson-Dirac GFLOP/s at the conventional 1320 flop per site per stencil application (BASELINE.json),
           value = 1320 * V * (2n+1) * steps * n_gpus / time; D_N applications per second and tau = time per Clenshaw
           iteration per site (the paper's normalisation) are reported alongside.
roofline = the dominant kernel (the Q stencil), timed alone with CUDA events on the launching stream in the same run
           (median of 5 batches, clocks sampled meanwhile), against the measured HBM copy peak of MEASURED_PEAKS.json;
           `q_kernel` holds every precision x recon variant and, for fp32, the stencil variants against each other.
layout   = a1 alone: pack / unpack / link compression, GB/s over AoS + SoA bytes.
next_rows = SURVEY 8(f): D_N^m inversion (fp64 CG, mixed precision), index by zero-mode counting, min-max coefficients.
projection = a7 alone: block dot and block axpy over l vectors (32^3x64 l = 8; 16^3x32 l = 50), GB/s over the compulsory bytes.
configs  = the other timed BASELINE.json configurations, driver-run in the same line: index 1 (1000 back-to-back Q on
           16^3x32, fp32 + fp64 x recon 12 / 8), index 3 (D_N on 8^3x16, fp64, about 20 modes from the library's
           eigen-solver) and index 4 (D_N on 16^3x32, fp32, about 50 modes, degree 200, eigen-solve timed).
cpu_baseline / --impl reference = the CPU oracle (oracle/, plain C + numpy, as it stands) on the host cores on a
           bounded sample of the same workload.

Multi-GPU: `--gpus N` splits the SAME 32^3x64 lattice along x0 over the N GPUs (domain decomposition,
csrc/shard.cu: two half-spinor faces per stencil over NCCL / NVLink, global reductions by all-reduce), scaling = strong;
`--replicas` runs N independent lattices instead (no data-path collective, scaling = weak).  When not started by torchrun the
script starts the N ranks itself.  Timing: barrier + synchronize, CUDA events, max over ranks.
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
QNORM = abs(4.0 + M_KERNEL) + 4.0


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


def kernel_source_sha16(kernel):
    """First 16 hex digits of the SHA-256 over the source files `kernel` is compiled from: what ties a row of the DRAM-traffic
    table to the code it was captured on (the GPU box has no .git).  A row whose hash differs from the current sources is
    reported as stale."""
    import hashlib

    files = ["wilson_tile.cu" if "tile" in kernel else "wilson.cu", "nd_dirac.cuh", "nd_su3.cuh"]
    h = hashlib.sha256()
    for f in files:
        with open(os.path.join(ROOT, "paper_1010_5636_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def load_traffic_row(kernel, lattice, prec, recon):
    """The row of profiles/q_kernel_dram_traffic.csv for exactly this kernel / lattice / precision / recon as a dict
    (bytes = dram__bytes_read.sum + dram__bytes_write.sum per launch from one ncu --set full capture, source_sha16 = the
    kernel sources it was captured on, capture = where the capture is summarised), or None."""
    p = os.path.join(ROOT, "profiles", "q_kernel_dram_traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            f_ = [s.strip() for s in line.split(",", 6)]
            if len(f_) >= 7 and f_[0] == kernel and f_[1] == lattice and f_[2] == str(prec) and f_[3] == str(recon):
                try:
                    return {"bytes": float(f_[4]), "source_sha16": f_[5], "capture": f_[6]}
                except ValueError:
                    return None
    return None


def load_traffic(kernel, lattice, prec, recon):
    """DRAM bytes per launch of `kernel` on `lattice` from the committed capture table, or None when there is no capture of
    exactly this kernel / lattice / precision / recon."""
    row = load_traffic_row(kernel, lattice, prec, recon)
    return None if row is None else row["bytes"]


def traffic_fields(kernel, lattice, prec, recon):
    """roofline keys about the DRAM traffic: the captured bytes, the sources they were captured on and whether those are the
    sources of this run."""
    row = load_traffic_row(kernel, lattice, prec, recon)
    cur = kernel_source_sha16(kernel)
    if row is None:
        return {"traffic": None, "traffic_source_sha16": None, "traffic_current_sha16": cur, "traffic_stale": None}
    return {"traffic": row["bytes"], "traffic_source_sha16": row["source_sha16"], "traffic_current_sha16": cur,
            "traffic_stale": row["source_sha16"] != cur, "traffic_capture": row["capture"]}


def stencil_kernel_name(variant, sites, prec=32):
    if variant == "tile":
        return "wilson_Q_tile2_kernel"
    if variant == "tile_tma":
        return "wilson_Q_tile3_kernel"
    if variant == "tile4":
        return "wilson_Q_tile_kernel"
    return "wilson_Q_hop_kernel" if sites < 16384 else "wilson_Q_kernel"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons every 200 ms while a timed region runs."""
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
            return self
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()
        return self

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
                "power_w_median": float(np.median(power)),
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
    """value = the units ALL ranks processed / the max-over-ranks time (replicas: every rank does units_per_rank; domain
    decomposition: units_per_rank is the rank's share of the one global lattice)."""
    return units_per_rank * world / (ms * 1e-3)


def spawn_command(argv, gpus, port):
    """The command line that starts `gpus` ranks of this script on one node (used when --gpus N > 1 is given without a
    torchrun environment)."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={gpus}", "--master-addr", "127.0.0.1",
            "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


# --------------------------------------------------------------------------------------------- CUDA arm
def build_modes(ctx, l, seed=99):
    """l orthonormal vectors and their Rayleigh quotients nu_k = <v_k, Q v_k> for the projection leg of the headline step
    (every call goes through the C ABI).  NOT eigenvectors: eq. 2.11 is defined for any orthonormal block and its cost
    does not depend on the values; the configs with real low modes (`configs`, --eigensolve) use nd_lowmodes_compute."""
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


def median_of_batches(torch, ctx, fn, reps, batches=5, warm=5):
    """CUDA events around `reps` repetitions after warm-up, median of `batches` batches -> ms per repetition."""
    for _ in range(warm):
        fn()
    t = [time_region(torch, ctx, fn, reps) / reps for _ in range(batches)]
    return float(np.median(t)), [float(x) for x in t]


def measure_q_kernel(torch, nd, dims, lattice, U64, prec, recon, peak, variants=(None,), reps=20):
    """The Q stencil alone: fixed source, separate destination, CUDA events on the launch stream."""
    ctx = nd.Context(dims, prec=prec, recon=recon, bc_time=-1)
    ctx.set_gauge(U64.astype(np.complex64) if prec == 32 else U64)
    x, y = ctx.new_spinor(), ctx.new_spinor()
    ctx.gaussian(x, 5636)
    V = ctx.V
    out = None
    for var in variants:
        if var is not None:
            try:
                ctx.set_stencil_variant(var)
            except nd.NDError:
                continue
        name = ctx.get_stencil_variant()
        ms, batches = median_of_batches(torch, ctx, lambda: ctx.apply_Q(y, x, M_KERNEL), reps)
        gbs = q_bytes_per_site(prec, recon) * V / (ms * 1e-3) / 1e9
        name = ctx.get_stencil_variant_for(False, 1)     # the dispatch's own choice for this call (auto depends on the call)
        kernel = stencil_kernel_name(name, V, prec)
        r = {"prec": prec, "recon": recon, "stencil_variant": name, "kernel": kernel, "us_per_launch": ms * 1e3,
             "us_per_launch_batches": [b * 1e3 for b in batches], "gflops_1320": FLOP_PER_SITE * V / (ms * 1e-3) / 1e9,
             "bytes_per_site": q_bytes_per_site(prec, recon), "achieved_gbs": gbs, "frac_of_measured_peak": gbs / peak,
             "frac_of_8TBs": gbs / 8000.0, "dram_traffic_ncu": load_traffic(kernel, lattice, prec, recon)}
        if out is None:
            out = r                      # the first variant is the one the library picks (auto)
            out["other_variants"] = {}
            # the same kernel with the Clenshaw update in its epilogue (a5: out = s0 Q(in) + s1 v1 + s2 v2 + s3 v3, out == v2):
            # every second stencil of a D_N application; three more vector streams in the byte model
            v = ctx.new_spinor(3)
            for j in range(3):
                ctx.gaussian(v[j], 77 + j)
            msf, _ = median_of_batches(torch, ctx, lambda: ctx.apply_Q_axpbycz(v[1], x, M_KERNEL, 0.05, -0.9, v[0], -0.5, v[1], 0.01, v[2]), reps)
            gbf = q_bytes_per_site(prec, recon, 3) * V / (msf * 1e-3) / 1e9
            out["fused_epilogue"] = {"kernel": stencil_kernel_name(ctx.get_stencil_variant_for(True, 1), V, prec),
                                     "us_per_launch": msf * 1e3, "bytes_per_site": q_bytes_per_site(prec, recon, 3),
                                     "achieved_gbs": gbf, "frac_of_measured_peak": gbf / peak, "frac_of_8TBs": gbf / 8000.0}
            del v
        else:
            out["other_variants"][name] = {k: r[k] for k in ("kernel", "us_per_launch", "achieved_gbs", "frac_of_measured_peak")}
    ctx.close()
    del x, y
    torch.cuda.empty_cache()
    return out


def sharded_probe(torch, nd, world, rank, local, p2p):
    """One stencil application on a tiny lattice split over the ranks (the transports bench.py is about to use), compared with
    the same lattice applied whole on this GPU: every site of the rank's part, and the global norm - which crosses the
    all-reduce and depends on both received faces - identical on all ranks by construction of the check."""
    from paper_1010_5636_b200.dist import make_comm

    gd = (4 * world, 4, 4, 8)
    U = gauge_field(gd, "smooth", eps=0.3)
    tb, tl, _, _ = nd.shard_layout(gd[0], world, rank)
    whole = nd.Context(gd, prec=64, recon=12, bc_time=-1, device=local)
    whole.set_gauge(U)
    x, y = whole.new_spinor(), whole.new_spinor()
    whole.gaussian(x, 99)
    whole.apply_Q(y, x, M_KERNEL)
    ref_norm, xa, ya = whole.norm2(y), whole.unpack_spinor(x), whole.unpack_spinor(y)
    part = nd.Context((tl,) + gd[1:], prec=64, recon=12, bc_time=-1, device=local)
    part.set_gauge(np.ascontiguousarray(U[:, tb:tb + tl]))
    comm, kind = make_comm(part, p2p=p2p)
    xl, yl = part.pack_spinor(np.ascontiguousarray(xa[tb:tb + tl])), part.new_spinor()
    part.apply_Q(yl, xl, M_KERNEL)
    got_norm = part.norm2(yl)
    err = float(np.abs(part.unpack_spinor(yl) - ya[tb:tb + tl]).max())
    part.close()
    whole.close()
    del comm
    if not (abs(got_norm - ref_norm) <= 1e-10 * ref_norm and err <= 1e-12 * np.sqrt(ref_norm)):
        raise RuntimeError(f"sharded stencil disagrees with the whole lattice: |y|^2 {got_norm} vs {ref_norm}, worst entry {err}")
    return kind


def measure_sustained(torch, nd, dims, U64, prec, recon, local, seconds=2.5):
    """The stencil variants where the D_N loop actually runs them (VERDICT r2 task 5): >= `seconds` of back-to-back launches,
    alternating the plain and the fused-epilogue stencil exactly as a Clenshaw step does, with clocks and board power sampled
    meanwhile.  A seconds-long loop sits at the power cap (~1.55 GHz instead of 1.9), so a variant that issues fewer
    instructions or draws less power can win here although it loses when timed alone at full clocks.  us_per_pair = one
    plain + one fused launch."""
    out = {}
    for var in ("auto", "site", "tile_tma") + (("tile4",) if prec == 32 else ()):
        ctx = nd.Context(dims, prec=prec, recon=recon, bc_time=-1, device=local)
        ctx.set_gauge(U64.astype(np.complex64) if prec == 32 else U64)
        try:
            ctx.set_stencil_variant(var)
        except nd.NDError:
            ctx.close()
            continue
        x, t = ctx.new_spinor(), ctx.new_spinor()
        v = ctx.new_spinor(3)
        ctx.gaussian(x, 1)
        for j in range(3):
            ctx.gaussian(v[j], 2 + j)

        def pair():
            ctx.apply_Q(t, x, M_KERNEL)
            ctx.apply_Q_axpbycz(v[1], t, M_KERNEL, 0.05, -0.9, v[0], -0.5, v[1], 0.01, v[2])   # bounded recurrence, out aliases v2

        for _ in range(20):
            pair()
        probe = time_region(torch, ctx, pair, 50) / 50                 # ms per pair at whatever the clocks are now
        reps = max(200, int(seconds * 1e3 / probe))
        sampler = ClockSampler(local).start()
        ms = time_region(torch, ctx, pair, reps)
        clocks = sampler.stop()
        out[var] = {"kernel_plain": stencil_kernel_name(ctx.get_stencil_variant_for(False, 1), ctx.V, prec),
                    "kernel_fused": stencil_kernel_name(ctx.get_stencil_variant_for(True, 1), ctx.V, prec),
                    "pairs": reps, "seconds": ms * 1e-3, "us_per_pair": ms * 1e3 / reps, "sm_mhz": clocks.get("sm_mhz"),
                    "power_w_median": clocks.get("power_w_median"), "power_w_max": clocks.get("power_w_max"),
                    "reasons": clocks.get("reasons")}
        ctx.close()
        del x, t, v
        torch.cuda.empty_cache()
    return out


def measure_layout(torch, nd, dims, U64, prec, peak):
    """a1 alone (VERDICT r1 task 6): AoS <-> SoA on the device, link compression; GB/s over the bytes of both sides."""
    ctx = nd.Context(dims, prec=prec, recon=12, bc_time=-1)
    with torch.cuda.stream(ctx.stream):
        aos = torch.view_as_complex(torch.randn(dims + (4, 3, 2), dtype=ctx.real_dtype, device=ctx.torch_device))
        back = torch.empty_like(aos)
        Ud = torch.from_numpy(U64.astype(np.complex64) if prec == 32 else U64).to(ctx.torch_device)
    soa = ctx.new_spinor()
    V, b = ctx.V, prec // 8
    res = {}
    ms, _ = median_of_batches(torch, ctx, lambda: ctx.lib.nd_pack_spinor(ctx._h, aos.data_ptr(), prec, 1, soa.data_ptr()), 20)
    res["pack_spinor"] = {"us": ms * 1e3, "gbs": 2 * 24 * b * V / (ms * 1e-3) / 1e9}
    ms, _ = median_of_batches(torch, ctx, lambda: ctx.lib.nd_unpack_spinor(ctx._h, soa.data_ptr(), back.data_ptr(), prec, 1), 20)
    res["unpack_spinor"] = {"us": ms * 1e3, "gbs": 2 * 24 * b * V / (ms * 1e-3) / 1e9}
    ctx.synchronize()
    res["round_trip_bit_exact"] = bool(torch.equal(aos, back))
    t = []
    for _ in range(4):                  # nd_set_gauge synchronises (it returns the SU(3) check): host clock around it
        ctx.synchronize()
        t0 = time.perf_counter()
        ctx.set_gauge(Ud)
        ctx.synchronize()
        t.append(time.perf_counter() - t0)
    ms = float(np.median(t[1:])) * 1e3
    res["set_gauge_recon12"] = {"us": ms * 1e3, "gbs": 4 * (18 + 12) * b * V / (ms * 1e-3) / 1e9,
                                "note": "host clock around the call (it synchronises to return the SU(3) check)"}
    for k in ("pack_spinor", "unpack_spinor", "set_gauge_recon12"):
        res[k]["frac_of_measured_peak"] = res[k]["gbs"] / peak
    res["prec"] = prec
    ctx.close()
    del aos, back, Ud, soa
    torch.cuda.empty_cache()
    return res


def measure_projection(torch, nd, lattice, l, prec, peak):
    """a7 alone: block dot (V^dagger x, l vectors) and block axpy (y += V a) through the `_dev` calls (no host synchronisation),
    GB/s over the compulsory bytes ((l + 1) resp. (l + 2) spinor streams)."""
    from lattice_inputs import parse_lattice

    dims = parse_lattice(lattice)
    ctx = nd.Context(dims, prec=prec, recon=12, bc_time=-1)
    V, b = ctx.V, prec // 8
    Vb, x = ctx.new_spinor(l), ctx.new_spinor()
    for k in range(l):
        ctx.gaussian(Vb[k], 300 + k)
    ctx.gaussian(x, 299)
    with torch.cuda.stream(ctx.stream):
        c = torch.zeros(2 * l, dtype=torch.float64, device=ctx.torch_device)
        a = torch.full((2 * l,), 1e-3, dtype=torch.float64, device=ctx.torch_device)
    reps = 20 if V * l < (1 << 26) else 5
    ms_dot, _ = median_of_batches(torch, ctx, lambda: ctx.block_dot_dev(Vb, x, c), reps)
    ms_axpy, _ = median_of_batches(torch, ctx, lambda: ctx.block_axpy_dev(a, Vb, x), reps)
    res = {"lattice": lattice, "prec": prec, "l": l, "block_bytes": l * 24 * b * V,
           "block_dot": {"us": ms_dot * 1e3, "gbs": (l + 1) * 24 * b * V / (ms_dot * 1e-3) / 1e9},
           "block_axpy": {"us": ms_axpy * 1e3, "gbs": (l + 2) * 24 * b * V / (ms_axpy * 1e-3) / 1e9}}
    for k in ("block_dot", "block_axpy"):
        res[k]["frac_of_measured_peak"] = res[k]["gbs"] / peak
    ctx.close()
    del Vb, x, c, a
    torch.cuda.empty_cache()
    return res


def measure_next_rows(torch, nd):
    """The SURVEY.md 8(f) rows beyond D_N itself, timed through the C ABI (parity of each is in tests/): f2 inversion of the massive
    operator D_N^m by CG on the normal equations in fp64 and with fp32 inner / fp64 outer refinement, f2 index by zero-mode
    counting on a constant-flux field, f4 min-max against interpolation coefficients (host utilities)."""
    from lattice_inputs import flux_su3, gauge_field

    res = {}
    # ---- f2: inversion on 8^3x16 (BASELINE config 3's lattice), no projected modes, quark mass 0.1
    dims, n, eps, mq = (16, 8, 8, 8), 100, 0.0045, 0.1
    U = gauge_field(dims, "smooth", eps=0.3)
    c, delta = nd.cheb_coeffs(n, eps)
    c64 = nd.Context(dims, prec=64, recon=12, bc_time=-1)
    c32 = nd.Context(dims, prec=32, recon=12, bc_time=-1)
    c64.set_gauge(U)
    c32.set_gauge(U.astype(np.complex64))
    for cc in (c64, c32):
        cc.set_sign_poly(c, eps, QNORM, M_KERNEL)
        cc.set_lowmodes(None, [])
    b, x = c64.new_spinor(), c64.new_spinor()
    c64.gaussian(b, 5636)
    c64.synchronize()
    t0 = time.perf_counter()
    relres, iters, ok = c64.solve_DNm(x, b, RHO, mq, tol=1e-8, maxit=400)
    c64.synchronize()
    t1 = time.perf_counter()
    relres_m, outer, inner, ok_m = c64.solve_DNm_mixed(c32, x, b, RHO, mq, tol=1e-8, inner_tol=1e-3)
    c64.synchronize()
    t2 = time.perf_counter()
    res["f2_inversion"] = {"lattice": "8^3x16", "degree": n, "eps": eps, "delta": delta, "quark_mass": mq, "tol": 1e-8,
                           "fp64_cg": {"seconds": t1 - t0, "iterations": iters, "relres": relres, "converged": ok,
                                       "sign_applications": 2 * iters + 2},
                           "mixed": {"seconds": t2 - t1, "outer_steps": outer, "fp32_cg_iterations": inner, "relres": relres_m,
                                     "converged": ok_m}}
    c64.close()
    c32.close()
    # ---- f2: index on a constant-flux field (|index| = 2 |q01 q23| = 2), low modes and sign function from the library
    dims = (8, 8, 4, 4)
    ctx = nd.Context(dims, prec=64, recon=12, bc_time=-1)
    ctx.set_gauge(flux_su3(dims, 1, 1, noise=0.05))
    ctx.synchronize()
    t0 = time.perf_counter()
    u, nu, resid, st = ctx.lowmodes_compute(2, M_KERNEL, tol=1e-8, maxit=80, lextra=6, degree=20, l_max=8, stop="residue")
    guard = float(np.abs(st["nu_guard"]).min())
    eps = 0.99 * guard ** 2 / QNORM ** 2
    c, delta = nd.cheb_coeffs(80, eps)
    ctx.set_sign_poly(c, eps, QNORM, M_KERNEL)
    ctx.set_lowmodes(u, nu)
    npl, nmi, ist = ctx.index_count(6, 1e-3, degree=8, maxit=40)
    ctx.synchronize()
    res["f2_index"] = {"lattice": "8x8x4x4 constant-flux field (q01 = q23 = 1, 5 % noise)", "n_plus": npl, "n_minus": nmi, "index": npl - nmi,
                       "seconds": time.perf_counter() - t0, "projected_modes": int(st["l_chosen"]), "sign_applications": ist["sign_applications"],
                       "lowest_nonzero": float(min(e for e in ist["evals"].ravel() if e > 1e-3))}
    ctx.close()
    # ---- f4: min-max (Remez) against interpolation coefficients at the headline's degree
    ci, di = nd.cheb_coeffs(100, 0.002)
    cm, dm, lev = nd.minmax_coeffs(100, 0.002)
    res["f4_minmax"] = {"degree": 100, "eps": 0.002, "delta_interpolation": di, "delta_minmax": dm, "levelled_error": lev}
    torch.cuda.empty_cache()
    return res


def dn_config(torch, nd, index, lattice, prec, field_eps, l_window, guard, n, eig_degree, bound_tol, nrhs, sources=10):
    """BASELINE.json configs[index]: D_N with the low modes from nd_lowmodes_compute (dynamic l, stop on the bound (2.10)),
    eps by DESIGN.md R11; D_N applications per second over `sources` Gaussian sources, single-source and batched."""
    from lattice_inputs import gauge_field, parse_lattice

    dims = parse_lattice(lattice)
    U = gauge_field(dims, "smooth", eps=field_eps)
    ctx = nd.Context(dims, prec=prec, recon=12, bc_time=-1)
    ctx.set_gauge(U.astype(np.complex64) if prec == 32 else U)
    V = ctx.V
    ctx.synchronize()
    t0 = time.perf_counter()
    modes, nu, resid, st = ctx.lowmodes_compute(l_window[0], M_KERNEL, tol=bound_tol, maxit=80, lextra=guard, degree=eig_degree,
                                                l_max=l_window[1], stop="bound")
    ctx.synchronize()
    eig_s = time.perf_counter() - t0
    eps = 0.99 * float((nu ** 2).max()) / QNORM ** 2
    c, delta = nd.cheb_coeffs(n, eps)
    ctx.set_sign_poly(c, eps, QNORM, M_KERNEL)
    ctx.set_lowmodes(modes, nu)
    eta, out, work = ctx.new_spinor(sources), ctx.new_spinor(sources), ctx.new_spinor(3)
    for j in range(sources):
        ctx.gaussian(eta[j], 5636 + j)

    def sweep():
        for j in range(sources):
            ctx.apply_DN(out[j], eta[j], 1.0 / RHO, work, use_graph=True)

    ms, _ = median_of_batches(torch, ctx, sweep, 1, batches=5, warm=2)
    r = {"config_index": index, "workload": f"D_N apply on {lattice}, exp({field_eps} i H) links, f{prec}, recon 12, degree n={n}, "
                                            f"low modes from nd_lowmodes_compute", "lattice": lattice, "sites": V,
         "dtype": f"f{prec}", "degree": n, "eps": eps, "delta": delta,
         "eigensolve": {"seconds": eig_s, "l_window": list(l_window), "guard": guard, "l_chosen": st["l_chosen"],
                        "stop": f"bound (2.10) <= {bound_tol}", "converged": st["converged"],
                        "outer_iterations": st["iterations"], "q_stencils": st["stencils"],
                        "max_residue_rho": float(resid.max()), "kappa_pm": [float(k) for k in st["kappa"]],
                        "projector_bound_pm": [float(b) if np.isfinite(b) else None for b in st["bound"]],
                        "nu2_min": float((nu ** 2).min()), "nu2_max": float((nu ** 2).max())},
         "sources": sources, "dn_applies_per_s": sources / (ms * 1e-3), "ms_per_dn": ms / sources,
         "gflops_1320": FLOP_PER_SITE * V * (2 * n + 1) * sources / (ms * 1e-3) / 1e9,
         "tau_ns_per_clenshaw_iteration_per_site": ms * 1e6 / sources / (n * V),
         "kernel": stencil_kernel_name(ctx.get_stencil_variant_for(True, 1), V, prec)}
    if nrhs > 1:
        nb = min(nrhs, sources)
        workb = ctx.new_spinor(3 * nb)
        ms_b, _ = median_of_batches(torch, ctx, lambda: ctx.apply_DN_multi(out[:nb], eta[:nb], 1.0 / RHO, workb, use_graph=True), 1,
                                    batches=5, warm=2)
        r["multi_rhs"] = {"nrhs": nb, "dn_applies_per_s": nb / (ms_b * 1e-3), "ms_per_batch": ms_b,
                          "tau_ns_per_clenshaw_iteration_per_site": ms_b * 1e6 / nb / (n * V)}
    ctx.close()
    del modes, eta, out, work
    torch.cuda.empty_cache()
    return r


def q_config(torch, nd, lattice="16^3x32", field_eps=0.3, reps=1000):
    """BASELINE.json configs[1]: 1000 back-to-back Q applications (fixed source, separate destination) on 16^3x32,
    fp32 and fp64 x recon 12 / 8.  The working set (<= 100 MB) is L2-resident: GFLOP/s and model GB/s, NOT an HBM fraction."""
    from lattice_inputs import gauge_field, parse_lattice

    dims = parse_lattice(lattice)
    U = gauge_field(dims, "smooth", eps=field_eps)
    runs = {}
    for prec, recon in ((32, 12), (32, 8), (64, 12), (64, 8)):
        ctx = nd.Context(dims, prec=prec, recon=recon, bc_time=-1)
        ctx.set_gauge(U.astype(np.complex64) if prec == 32 else U)
        x, y = ctx.new_spinor(), ctx.new_spinor()
        ctx.gaussian(x, 5636)
        f = lambda: ctx.apply_Q(y, x, M_KERNEL)
        for _ in range(10):
            f()
        ms = time_region(torch, ctx, f, reps)
        V = ctx.V
        runs[f"f{prec}_recon{recon}"] = {"ms_for_1000": ms, "us_per_Q": ms * 1e3 / reps,
                                         "gflops_1320": FLOP_PER_SITE * V * reps / (ms * 1e-3) / 1e9,
                                         "model_gbs": q_bytes_per_site(prec, recon) * V * reps / (ms * 1e-3) / 1e9,
                                         "kernel": stencil_kernel_name(ctx.get_stencil_variant_for(False, 1), V, prec)}
        ctx.close()
        del x, y
    torch.cuda.empty_cache()
    return {"config_index": 1, "workload": f"{reps} back-to-back Q on {lattice}, exp({field_eps} i H) links, m=-1.6", "lattice": lattice,
            "note": "working set is L2-resident: GFLOP/s and byte-model GB/s, not an HBM-roofline fraction", "runs": runs}


# ------------------------------------------------------------------------------------------ CPU oracle legs
def oracle_q_alone(lattice, reps=2):
    """Seconds per Q of the plain-C oracle (oracle/wilson_ref.c, fp64, full 3x3 links) with the OpenMP threads the
    environment gives it (run in a subprocess to fix OMP_NUM_THREADS)."""
    from lattice_inputs import gauge_field, gaussian_spinor, parse_lattice
    from oracle import wilson_c

    dims = parse_lattice(lattice)
    sd = tuple(min(d, 8) for d in dims)            # a periodic 8^4 Haar block tiled over the lattice: same cost, quick to draw
    small = gauge_field(sd, "haar")
    U = np.tile(small, (1,) + tuple(d // e for d, e in zip(dims, sd)) + (1, 1))
    psi = gaussian_spinor(dims)
    Q = wilson_c.make_Q(U, M_KERNEL, -1)
    Q(psi)
    t0 = time.perf_counter()
    for _ in range(reps):
        Q(psi)
    dt = (time.perf_counter() - t0) / reps
    return {"lattice": lattice, "threads": wilson_c.num_threads(), "seconds_per_Q": dt,
            "gflops_1320": FLOP_PER_SITE * int(np.prod(dims)) / dt / 1e9}


def oracle_q_alone_subprocess(lattice, threads):
    env = dict(os.environ)
    if threads:
        env["OMP_NUM_THREADS"] = str(threads)
    code = f"import sys, json; sys.path.insert(0, {ROOT!r}); import bench; print(json.dumps(bench.oracle_q_alone({lattice!r})))"
    try:
        r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=300)
        return json.loads(r.stdout.strip().splitlines()[-1])
    except Exception as e:          # the baseline is context: never let it take the line down
        return {"lattice": lattice, "threads": threads, "error": str(e)[:200]}


def cpu_baseline_sample(steps=1, n=10, l=2, dims=(64, 32, 32, 32), U=None):
    """The oracle as it stands on the host cores: its D_N recipe (oracle/sign.py eq. 2.11 + 2.4 over the plain-C stencil
    oracle/wilson_ref.c, fp64, full 3x3 links) on a bounded sample of the line's own workload: the SAME lattice and field
    recipe, a lower polynomial degree n and l orthonormal projection vectors (10-30 s of CPU work per step)."""
    from lattice_inputs import gauge_field, gaussian_spinor
    from oracle import lowmodes as olow
    from oracle import sign as osign
    from oracle import wilson, wilson_c

    if U is None:
        U = gauge_field(dims, "haar")
    eta = gaussian_spinor(dims)
    Q = wilson_c.make_Q(U, M_KERNEL, -1)
    eps = 0.002
    c = osign.cheb_coeffs(n, eps)
    rng = np.random.Generator(np.random.PCG64(3))
    Vs = olow.orthonormalise([rng.standard_normal(eta.shape) + 1j * rng.standard_normal(eta.shape) for _ in range(l)])
    nu, Us = osign.rayleigh_ritz_Q(Q, Vs)
    osign.apply_DN(Q, wilson.apply_gamma5, eta, c[:2], eps, QNORM, 1.0 / RHO, nu, Us)    # warm-up (loads the C library)
    t0 = time.perf_counter()
    for _ in range(steps):
        osign.apply_DN(Q, wilson.apply_gamma5, eta, c, eps, QNORM, 1.0 / RHO, nu, Us)
    dt = (time.perf_counter() - t0) / steps
    vol = int(np.prod(dims))
    gflops = FLOP_PER_SITE * vol * (2 * n + 1) / dt / 1e9
    return {"value": gflops, "unit": "GFLOP/s", "cores": wilson_c.num_threads(), "kind": "oracle", "cpu_model": cpu_model(),
            "sample": f"oracle D_N recipe (oracle/sign.py over oracle/wilson_ref.c, fp64, full 3x3 links) on a "
                      f"{dims[1]}^3x{dims[0]} Haar lattice at degree n={n}, l={l} (synthetic orthonormal vectors): "
                      f"{2 * n + 1} stencils/step, {dt:.2f} s/step",
            "dn_applies_per_s": 1.0 / dt, "seconds_per_step": dt,
            "tau_ns_per_clenshaw_iteration_per_site": dt * 1e9 / (n * vol)}


# ---------------------------------------------------------------------------------------------- main arms
def run_b200(args):
    import torch

    import paper_1010_5636_b200 as nd
    from lattice_inputs import gauge_field, parse_lattice

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the CUDA path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    gdims = parse_lattice(args.lattice)
    prec, recon, n, l = args.prec, args.recon, args.degree, args.lowmodes
    peak, peak_src = load_peaks()

    # BASELINE config index 2: Haar-random links, seeded (--field smooth for the exp(i eps H) recipe)
    U64 = gauge_field(gdims, args.field, eps=args.field_eps)
    decompose = world > 1 and not args.replicas
    comm_kind, shard_fallback = None, None
    if decompose:
        # Before anything is sized for the decomposition: one tiny sharded stencil checked against the same lattice on this GPU
        # alone, the verdict agreed between the ranks.  If the transports cannot be set up here (or give wrong faces), the run
        # falls back to N independent replicas and says so, rather than hanging or failing in the headline path.
        from paper_1010_5636_b200.dist import CommSetupError, run_agreed

        try:
            run_agreed(lambda: sharded_probe(torch, nd, world, rank, local, args.p2p), "sharded probe",
                       torch.device("cuda", local))
        except CommSetupError as e:
            shard_fallback = str(e)
            decompose = False
            if rank == 0:
                print(f"bench.py: domain decomposition unavailable ({e}); running {world} replicas instead", file=sys.stderr)
    if decompose:
        # domain decomposition: this rank's time-slices of the one global lattice (nd_shard_layout), faces over NCCL
        from paper_1010_5636_b200.dist import make_comm

        tb, tl, _, _ = nd.shard_layout(gdims[0], world, rank)
        dims = (tl,) + tuple(gdims[1:])
        Uloc = np.ascontiguousarray(U64[:, tb:tb + tl])
    else:
        dims, Uloc = gdims, U64
    if args.sustained:
        # the variants inside a seconds-long loop at the power cap (rank 0's GPU; one JSON line, not the bench line)
        if rank == 0:
            print(json.dumps({"sustained": measure_sustained(torch, nd, gdims, U64, prec, recon, local, seconds=args.sustained),
                              "lattice": args.lattice, "prec": prec, "recon": recon}))
        return
    if args.q_only:
        # the stencil of one precision / recon alone (the command the ncu captures under profiles/ run)
        variants = (None,) if args.variant is None else (args.variant,)
        r = measure_q_kernel(torch, nd, gdims, args.lattice, U64, prec, recon, peak, variants, reps=args.steps)
        print(json.dumps({"q_only": r, "lattice": args.lattice, "peak_gbs": peak, "peak_source": peak_src}))
        return
    # the dominant kernel of the line's own precision / recon ALONE, before the long D_N legs heat the GPU into its power cap
    # (rank 0; the roofline object below is built from this leg)
    main_q, main_q_clocks = None, None
    if rank == 0:
        qs = ClockSampler(local).start()
        main_q = measure_q_kernel(torch, nd, gdims, args.lattice, U64, prec, recon, peak,
                                  (None, "site", "tile_tma", "tile4") if prec == 32 else (None, "site", "tile_tma"))
        main_q_clocks = qs.stop()
    ctx = nd.Context(dims, prec=prec, recon=recon, bc_time=-1, device=local)
    ctx.set_gauge(Uloc.astype(np.complex64) if prec == 32 else Uloc)
    # from here on every call acts on the global lattice; --p2p: faces stored by the pack kernel into the neighbours' windows
    comm = None
    if decompose:
        comm, comm_kind = make_comm(ctx, p2p=args.p2p)    # (p2p falls back to NCCL send/recv with the reason on stderr)
    V = ctx.V                                             # sites of this rank
    c, delta = nd.cheb_coeffs(n, args.eps)
    ctx.set_sign_poly(c, args.eps, QNORM, M_KERNEL)
    eig = None
    modes_kind = "synthetic orthonormal vectors with their Rayleigh quotients (not eigenvectors; eps not tied to the spectrum)"
    if args.eigensolve and l > 0:
        ctx.synchronize()
        t0 = time.perf_counter()
        modes, nu, resid, st = ctx.lowmodes_compute(max(1, l - l // 8), M_KERNEL, tol=args.eig_tol, maxit=60, lextra=max(8, l // 4),
                                                    degree=args.eig_degree, l_max=l + l // 8, stop="bound")
        ctx.synchronize()
        l = st["l_chosen"]
        eig = {"seconds": time.perf_counter() - t0, "l_chosen": l, "tol_bound_2_10": args.eig_tol, "converged": st["converged"],
               "outer_iterations": st["iterations"], "q_stencils": st["stencils"], "max_residue_rho": float(resid.max()),
               "kappa_pm": [float(k) for k in st["kappa"]],
               "projector_bound_pm": [float(b) if np.isfinite(b) else None for b in st["bound"]],
               "nu2_min": float((nu ** 2).min()), "nu2_max": float((nu ** 2).max())}
        args.eps = 0.99 * float((nu ** 2).max()) / QNORM ** 2
        c, delta = nd.cheb_coeffs(n, args.eps)
        ctx.set_sign_poly(c, args.eps, QNORM, M_KERNEL)
        modes_kind = "nd_lowmodes_compute (dynamic l, bound (2.10)); eps by DESIGN.md R11"
    else:
        modes, nu = build_modes(ctx, l)
    ctx.set_lowmodes(modes, nu)
    eta, out, work = ctx.new_spinor(), ctx.new_spinor(), ctx.new_spinor(3)
    ctx.gaussian(eta, 5636 + (0 if decompose else rank))  # replicas: a different source per rank
    step = lambda: ctx.apply_DN(out, eta, 1.0 / RHO, work, use_graph=True)   # (no graph while sharded: host callbacks)

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
    headline_variant = ctx.get_stencil_variant()

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
    ms_e2e_serial = time_region(torch, ctx, e2e_step, args.steps)
    ms_e2e_serial = max_over_ranks(ms_e2e_serial, world, torch.device("cuda", local))
    hbytes = V * 24 * (prec // 8)

    # the same K steps as a user with a stream of sources would issue them: a second context of the same lattice on its own
    # stream does the layout calls (H2D + pack of source i+1, unpack + D2H of result i-1) while the operator works on source i;
    # every step still copies its own input in and its own result out, all through the C ABI
    io = nd.Context(dims, prec=prec, recon=recon, bc_time=-1, device=local)
    eta2, out2 = [eta, ctx.new_spinor()], [out, ctx.new_spinor()]
    ev_in = [torch.cuda.Event() for _ in range(2)]
    ev_out = [torch.cuda.Event() for _ in range(2)]

    def e2e_pipelined(k):
        io.pack_spinor_host(h_in.data_ptr(), prec, eta2[0])
        ev_in[0].record(io.stream)
        for i in range(k):
            b = i % 2
            ctx.stream.wait_event(ev_in[b])
            ctx.apply_DN(out2[b], eta2[b], 1.0 / RHO, work, use_graph=not decompose)
            ev_out[b].record(ctx.stream)
            if i > 0:
                io.stream.wait_event(ev_out[1 - b])           # result i-1 is complete, and source buffer 1-b is free again
                if i + 1 < k:
                    io.pack_spinor_host(h_in.data_ptr(), prec, eta2[1 - b])
                    ev_in[1 - b].record(io.stream)
                io.unpack_spinor_host(out2[1 - b], h_out.data_ptr(), prec)    # synchronises the io stream (host result)
            elif k > 1:
                io.pack_spinor_host(h_in.data_ptr(), prec, eta2[1])
                ev_in[1].record(io.stream)
        io.stream.wait_event(ev_out[(k - 1) % 2])
        io.unpack_spinor_host(out2[(k - 1) % 2], h_out.data_ptr(), prec)

    e2e_pipelined(2)
    ctx.synchronize()
    if world > 1:
        dist.barrier()
    t0e = torch.cuda.Event(enable_timing=True)
    t1e = torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t0e.record(io.stream)
    e2e_pipelined(args.steps)
    ctx.synchronize()
    t1e.record(io.stream)
    io.synchronize()
    ms_e2e = max_over_ranks(t0e.elapsed_time(t1e), world, torch.device("cuda", local))
    e2e_value = whole_job_value(gflop_per_step * args.steps, world, ms_e2e)
    io.close()

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return
    # ---- rank 0 only: the dominant kernel alone (roofline), every variant; layout; the other configs; the CPU oracle
    # (single-GPU legs on the global lattice; the other ranks wait at the final barrier)
    ctx.close()
    del modes, eta, out, work, comm, eta2, out2
    torch.cuda.empty_cache()
    dims = gdims
    V_global = int(np.prod(gdims))
    qk = {f"f{prec}_recon{recon}": main_q}
    for p, r in ((32, 12), (64, 12), (32, 8), (64, 8), (32, 18), (64, 18)):
        if (p, r) == (prec, recon) or args.quick:
            continue
        variants = (None, "site", "tile_tma", "tile4") if p == 32 else (None, "site", "tile_tma")
        qk[f"f{p}_recon{r}"] = measure_q_kernel(torch, nd, gdims, args.lattice, U64, p, r, peak, variants)
    q_clocks = main_q_clocks
    main = main_q
    # the same kernel in the other precision (north star: ">= 70 % of HBM bandwidth in fp32 AND fp64"): inside `roofline`, so that
    # a record which keeps only the contract's keys carries both precisions
    oprec = 64 if prec == 32 else 32
    okey = f"f{oprec}_recon12"
    if okey not in qk:
        qk[okey] = measure_q_kernel(torch, nd, gdims, args.lattice, U64, oprec, 12, peak, (None,))
    other = qk[okey]
    okern = other["kernel"]
    roofline = {"bound": "hbm", "achieved": main["achieved_gbs"], "peak": peak, "unit": "GB/s",
                "frac": main["achieved_gbs"] / peak,
                **traffic_fields(main["kernel"], args.lattice, prec, recon),
                f"fp{oprec}": {"kernel": f"{okern} (Q stencil, plain epilogue, recon 12)", "achieved": other["achieved_gbs"], "peak": peak,
                               "unit": "GB/s", "frac": other["achieved_gbs"] / peak, "frac_of_8TBs_nominal": other["achieved_gbs"] / 8000.0,
                               "us_per_launch": other["us_per_launch"], "us_per_launch_batches": other["us_per_launch_batches"],
                               "algorithmic_bytes_per_launch": other["bytes_per_site"] * V_global,
                               **traffic_fields(okern, args.lattice, oprec, 12),
                               "fused_epilogue": other.get("fused_epilogue")},
                "kernel": f"{main['kernel']} (Q stencil, plain epilogue; stencil variant '{main['stencil_variant']}')",
                "peak_source": peak_src, "algorithmic_bytes_per_launch": main["bytes_per_site"] * V_global,
                "us_per_launch": main["us_per_launch"],
                "timing": "median of 5 batches of 20 launches, CUDA events on the launch stream; first leg of the run (before the D_N legs)",
                "frac_of_8TBs_nominal": main["achieved_gbs"] / 8000.0, "clocks": q_clocks,
                "traffic_source": "profiles/q_kernel_dram_traffic.csv (ncu --set full of this kernel on this lattice; null = no capture; "
                                  "traffic_stale = the kernel's sources have changed since the capture)"}
    layout, projection, configs, cpu, next_rows = None, None, [], None, None
    if not args.quick:
        layout = {f"f{p}": measure_layout(torch, nd, dims, U64, p, peak) for p in (32, 64)}
        projection = [measure_projection(torch, nd, "32^3x64", 8, 32, peak), measure_projection(torch, nd, "16^3x32", 50, 32, peak),
                      measure_projection(torch, nd, "16^3x32", 50, 64, peak)]
        configs.append(q_config(torch, nd))
        configs.append(dn_config(torch, nd, 3, "8^3x16", 64, 0.3, (16, 24), 8, 100, 60, 1e-6, nrhs=10))
        configs.append(dn_config(torch, nd, 4, "16^3x32", 32, 0.25, (44, 56), 12, 200, 160, 1e-2, nrhs=4))
        next_rows = measure_next_rows(torch, nd)
    if not args.no_cpu_baseline and not args.quick:
        cpu = cpu_baseline_sample(dims=dims, U=U64)
        ncores = os.cpu_count() or 1
        cpu["q_alone"] = [oracle_q_alone_subprocess(lat, th) for lat in ("16^3x32", "32^3x64") for th in (1, ncores)]
        # the oracle's D_N on the lattices of BASELINE configs 3 and 4 (SURVEY.md 8(d) "CPU baseline"): the full degree of config 3,
        # a bounded degree and fewer vectors for config 4 (its full n = 200, l = 50 would take minutes in numpy)
        from lattice_inputs import gauge_field as _gf

        cpu["dn_configs"] = []
        for idx, cd, feps, cn, cl in ((3, (16, 8, 8, 8), 0.3, 100, 8), (4, (32, 16, 16, 16), 0.25, 40, 4)):
            r = cpu_baseline_sample(n=cn, l=cl, dims=cd, U=_gf(cd, "smooth", eps=feps))
            cpu["dn_configs"].append({"config_index": idx, "lattice": f"{cd[1]}^3x{cd[0]}", "degree": cn, "vectors": cl, "cores": r["cores"],
                                      "seconds_per_dn": r["seconds_per_step"], "gflops_1320": r["value"],
                                      "tau_ns_per_clenshaw_iteration_per_site": r["tau_ns_per_clenshaw_iteration_per_site"]})
    elif not args.no_cpu_baseline:
        cpu = cpu_baseline_sample(dims=(32, 16, 16, 16), n=6)
    line = {
        "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong" if decompose else "weak", "vs_baseline": None,
        "dtype": "f32" if prec == 32 else "f64", "data": "synthetic",
        "config": {"workload": f"D_N apply (eq. 2.4+2.11) on {args.lattice}, {args.field} SU(3) links, m=-1.6, recon {recon}, "
                               f"degree n={n} (2n+1={stencils} Q stencils), l={l} projected vectors, CUDA graph",
                   "lattice": args.lattice, "sites": V_global, "sites_per_gpu": V, "recon": recon, "degree": n, "eps": args.eps,
                   "delta": delta, "lowmodes": l, "lowmodes_kind": modes_kind, "stencil_variant": headline_variant,
                   "parallelism": (f"domain decomposition along x0 over {world} GPUs ({gdims[0] // world} slices each), "
                                   f"half-spinor faces {'stored peer-to-peer into symmetric memory' if comm_kind == 'p2p' else 'over NCCL'}"
                                   if decompose else f"replicas x{world}" + (f" (fallback: {shard_fallback})" if shard_fallback else "")),
                   "l2_policy": "inputs larger than L2 (links + vectors >= 1.4 GB fp32), no flush needed"},
        "dn_applies_per_s": (1 if decompose else world) * args.steps / (ms * 1e-3),
        "q_stencils_per_s": (1 if decompose else world) * args.steps * stencils / (ms * 1e-3),
        "tau_ns_per_clenshaw_iteration_per_site": ms * 1e6 / args.steps / (n * V * (world if decompose else 1)),
        "tau_paper_ns": {"single_GTX285": 38.0, "double_GTX285": 90.0, "source": "PAPER.md:L140-142 (context, other hardware)"},
        "e2e": {"value": e2e_value, "unit": "GFLOP/s", "h2d_bytes_per_step": hbytes, "d2h_bytes_per_step": hbytes,
                "ms_per_step": ms_e2e / args.steps,
                "how": "pinned host AoS -> nd_pack_spinor (H2D) -> nd_apply_DN -> nd_unpack_spinor (D2H) every step; the layout calls of "
                       "steps i+1 / i-1 run on a second context's stream while the operator works on step i",
                "serial_ms_per_step": ms_e2e_serial / args.steps,
                "serial_value": whole_job_value(gflop_per_step * args.steps, world, ms_e2e_serial)},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": roofline,
        "q_kernel": qk,
        "layout": layout,
        "projection": projection,
        "next_rows": next_rows,
        "configs": configs,
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
    # W warm-up + K timed steps of the oracle, each step one D_N application on a bounded sample of the CUDA arm's workload
    # (same field recipe and operator; a 16^3x32 lattice at degree 40 keeps a K-step run within minutes on the host cores)
    dims = (32, 16, 16, 16)
    from lattice_inputs import gauge_field

    U = gauge_field(dims, "haar")
    cpu_baseline_sample(steps=max(args.warmup, 1), n=1, l=4, dims=dims, U=U)
    r = cpu_baseline_sample(steps=args.steps, n=40, l=4, dims=dims, U=U)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": "GFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["seconds_per_step"] * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "CPU oracle: " + r["sample"]},
        "cpu_baseline": {"value": r["value"], "unit": "GFLOP/s", "kind": "oracle", "cores": r["cores"], "sample": r["sample"],
                         "cpu_model": r["cpu_model"]},
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
    ap.add_argument("--eig-degree", type=int, default=100)
    ap.add_argument("--quick", action="store_true", help="headline + its own Q-kernel variant only (no layout / configs legs)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--q-only", action="store_true", help="time only the Q stencil of --prec / --recon on --lattice (plain and fused epilogue)")
    ap.add_argument("--variant", default=None, choices=["site", "tile", "tile_tma", "tile4"], help="with --q-only: force a stencil variant")
    ap.add_argument("--sustained", type=float, default=0.0, metavar="SECONDS",
                    help="time every stencil variant in a loop of alternating plain / fused launches of at least SECONDS each, "
                         "with clocks and power sampled (the regime of the D_N step), print one JSON line and exit")
    ap.add_argument("--p2p", action="store_true", help="--gpus N: peer-to-peer face exchange (dist.PeerComm) instead of NCCL send/recv")
    ap.add_argument("--replicas", action="store_true", help="--gpus N as N independent lattices (weak scaling) instead of the domain decomposition")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started as `python bench.py --gpus N`: start the N ranks ourselves (one per GPU, NCCL only for the barrier)
        import socket

        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        raise SystemExit(subprocess.call(spawn_command(sys.argv[1:], args.gpus, port)))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
