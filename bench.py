#!/usr/bin/env python
"""bench.py -- the BASELINE.json metric on one B200 (or N independent replicas under torchrun).

Metric (BASELINE.json): "Dslash ns/site and HBM GB/s (fraction of peak), 1xB200 double; mshift-CG s/iter".

  step      one iteration of the multi-shift CG = one pass of the whole hot path (DESIGN.md rows A2-A9:
            D_oe, D_eo + fused zaxpy/dot epilogue, scalar recurrences, residual update + norm, x_i/p_i
            updates of every active shift, loop control); A1 (link storage) is one-time set-up.
  workload  BASELINE config 4: 48^4, 16 shifts geometric 1e-5..1, m = 0.0075, tol 1e-10, 18-real links,
            seeded random SU(3) links + Gaussian even-site source (lqcd_inputs).  Links (3.06 GB) are far
            larger than L2, so no explicit L2 flush is needed between iterations.
  value     seconds per CG iteration over exactly K iterations (device time, CUDA events), inputs
            resident in HBM.  `dslash` holds ns/site and GB/s of the operator alone at 32^4 and 48^4,
            18- and 12-real links; `roofline` is the D_oe/D_eo kernel at 48^4 (18-real) against the
            measured HBM copy bandwidth; `full_solve` is the same solve run to convergence.
  e2e       the same K iterations through lqcd_mshift_cg_host: b read from pinned host memory, all 16
            solutions written back to pinned host memory, copies inside the timed region.
  cpu_baseline  the CPU oracle (oracle/, as it stands) timed on the host cores on a few iterations of the
            same workload.  `--impl reference` runs only that.

Usage:  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

import lqcd_inputs as gen  # noqa: E402

# Algorithmic bytes, per output site of one parity application.
DSLASH_BYTES = {18: 8 * 144 + 8 * 48 + 48, 12: 8 * 96 + 8 * 48 + 48}      # 1584 / 1200
DSLASH_DRAM_MODEL = {18: 8 * 144 + 48 + 48, 12: 8 * 96 + 48 + 48}         # each input read from DRAM once
DSLASH_FLOPS = {18: 570, 12: 570 + 8 * 42}

# DRAM bytes per launch of dslash_kernel<18,0> measured by `ncu --set full` (dram__bytes_read.sum +
# dram__bytes_write.sum), keyed by workload; source file under profiles/.  None until captured.
NCU_DRAM_BYTES_PER_LAUNCH = {
    ("config4_48^4", 18): 3.190834e9 + 0.103419e9,     # profiles/ncu_full_r01.md, dslash_kernel<double,18,0>
    ("config4_48^4", 12): 2.171204e9 + 0.101689e9,     # profiles/ncu_full_r01.md, dslash_kernel<double,12,0>
}


def cg_bytes_per_site(n_active: int, recon: int) -> int:
    """SURVEY.md §8(d) model of one CG iteration per even site, shift updates applied every iteration:
    two Dslash + p in the epilogue + r update + base x/p + 192 B per further active shift."""
    return 2 * DSLASH_BYTES[recon] + 48 + 144 + 240 + 192 * (n_active - 1)


def cg_bytes_moved(freeze_iter, iters: int, m: int, recon: int) -> int:
    """Bytes per even site the library actually moves in `iters` iterations with block-deferred shift updates
    (DESIGN.md "CG iteration"): per iteration two Dslash + p (48) + r update (144) + base x/p (240); per block of
    m iterations one sweep reading the block's residuals (48 each) and updating x_i, p_i (192) of every shifted
    system that was active when the block began."""
    base = max(range(len(freeze_iter)), key=lambda i: freeze_iter[i])
    total = iters * (2 * DSLASH_BYTES[recon] + 48 + 144 + 240)
    for n0 in range(0, iters, m):
        nres = min(m, iters - n0)
        n_in = sum(1 for i, fz in enumerate(freeze_iter) if i != base and fz > n0)
        if n_in:
            total += 48 * nres + 192 * n_in
    return total


_T0 = time.perf_counter()


def phase(name: str):
    """wall-clock phase marks on stderr (BENCH_TIMING=1), to keep the default run within a few minutes"""
    if os.environ.get("BENCH_TIMING"):
        print(f"[bench {time.perf_counter() - _T0:7.1f} s] {name}", file=sys.stderr, flush=True)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU while the timed region runs (pynvml thread)."""

    def __init__(self, index: int, period: float = 0.02):
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                try:
                    phys = int(vis.split(",")[index])
                except Exception:
                    phys = index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def dist_setup(n_gpus: int):
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        if torch.cuda.is_available():
            torch.cuda.set_device(local)
        dist.init_process_group(backend=backend)
    return world, rank, local


def barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(world, value: float) -> float:
    if world == 1:
        return value
    import torch.distributed as dist
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    t = torch.tensor([value], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_replicas(world: int, local_ms_total: float, steps: int):
    """N independent replicas: the timed region lasts as long as the slowest rank; in that
    time the job advanced world*steps iterations.  Returns (ms_per_step of one replica, aggregate s/iter)."""
    ms_total = max_over_ranks(world, local_ms_total)
    ms_step = ms_total / steps
    return ms_total, ms_step, ms_step * 1e-3 / world


def sum_over_ranks(world, value: float) -> float:
    if world == 1:
        return value
    import torch.distributed as dist
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    t = torch.tensor([value], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def time_dslash(lq, L, recon, reps, warm, links=None, field=None, slab=None):
    """ns/site and GB/s of one parity application: reps x (D_oe: b->t, D_eo: t->u) with fixed b
    (never fed back: |D| ~ 2.6 on random links would overflow).  slab = (L_global, rank, nranks): the same on a slab
    context (two face exchanges over NCCL, interior and border launches per application); collective."""
    U = links if links is not None else gen.random_su3_links(L, device="cuda")
    f = field if field is not None else gen.gaussian_field(L, device="cuda")
    lat = lq.Lattice(L, recon=recon) if slab is None else lq.Lattice(slab[0], recon=recon, slab=slab[1:], comm="nccl")
    lat.set_gauge(U)
    b = lat.pack(f, 0)
    t = torch.empty_like(b)
    u = torch.empty_like(b)
    for _ in range(warm):
        lat.doe(b, out=t)
        lat.deo(t, out=u)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.current_stream().synchronize()
    n0 = lat.launches
    e0.record()
    for _ in range(reps):
        lat.doe(b, out=t)
        lat.deo(t, out=u)
    e1.record()
    torch.cuda.current_stream().synchronize()
    launches = lat.launches - n0
    ms = e0.elapsed_time(e1) / (2 * reps)
    lat.close()
    ns_site = ms * 1e6 / lat.Vh
    return {"us_per_application": ms * 1e3, "ns_per_site": ns_site,
            "gbs_algorithmic": DSLASH_BYTES[recon] / ns_site,
            "gbs_dram_model": DSLASH_DRAM_MODEL[recon] / ns_site,
            "gflops": DSLASH_FLOPS[recon] / ns_site, "launches": launches,
            "bytes_per_launch": DSLASH_BYTES[recon] * lat.Vh}


def read_only_reference_gbs():
    """Context for the roofline: what a plain read-only stream reaches on this GPU (torch.sum over 4 GiB of doubles,
    best of 10, CUDA events).  The measured peak of MEASURED_PEAKS.json is a COPY (half writes); the Dslash is 97 %
    reads."""
    a = torch.ones(1 << 29, dtype=torch.float64, device="cuda")
    best = 0.0
    for i in range(13):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        a.sum()
        e1.record()
        torch.cuda.current_stream().synchronize()
        if i >= 3:
            best = max(best, a.numel() * 8 / (e0.elapsed_time(e1) * 1e6))
    del a
    return best


def time_next_rows(lq, L, mass, shifts, tol, K, W, U, f):
    """The widened rows on the same workload, K iterations / applications each, device time:
    NEXT-1 rational sum, NEXT-2 single precision (Dslash and CG), NEXT-4 general U(1) phases (Dslash)."""
    res = {}
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def dslash_ns(lat, b, reps=max(K // 2, 20)):
        t, u = torch.empty_like(b), torch.empty_like(b)
        for _ in range(5):
            lat.doe(b, out=t)
            lat.deo(t, out=u)
        e0, e1 = ev(), ev()
        torch.cuda.current_stream().synchronize()
        e0.record()
        for _ in range(reps):
            lat.doe(b, out=t)
            lat.deo(t, out=u)
        e1.record()
        torch.cuda.current_stream().synchronize()
        return e0.elapsed_time(e1) * 1e6 / (2 * reps) / lat.Vh

    def cg_s_per_iter(lat, solve):
        lat.set_option(lq.LQCD_OPT_MAX_ITER, max(W, 3))
        solve()
        lat.set_option(lq.LQCD_OPT_MAX_ITER, K)
        info = solve()
        return info["solve_ms"] * 1e-3 / max(info["iters"], 1), info["iters"]

    # NEXT-1 and NEXT-4 on a double-precision context
    lat = lq.Lattice(L, mass=mass)
    lat.set_gauge(U)
    b = lat.pack(f, 0)
    alpha = [1.0 / (1 + i) for i in range(len(shifts))]
    y = torch.empty_like(b)
    s_it, n = cg_s_per_iter(lat, lambda: lat.rational_apply(b, 0.5, alpha, shifts, tol, y=y, raise_on_noconv=False)[1])
    res["next1_rational_apply"] = {"s_per_iter": s_it, "iters": n,
                                   "note": "y = alpha0 b + sum_i alpha_i x_i accumulated in the solve, x_i never stored"}
    theta = gen.random_u1_phases(L, device="cuda")
    lat.set_u1_phases(theta)
    ns = dslash_ns(lat, b)
    res["next4_u1_dslash"] = {"ns_per_site": ns, "gbs_algorithmic": (DSLASH_BYTES[18] + 64) / ns,
                              "gbs_dram_model": (DSLASH_DRAM_MODEL[18] + 64) / ns,
                              "note": "18-real links + theta_mu(x) (8 B/link), sincos in the kernel"}
    lat.close()
    del theta, y
    # NEXT-2: single precision
    lat = lq.Lattice(L, mass=mass, precisions=lq.LQCD_PREC_F32)
    lat.set_gauge(U)
    b32 = b.float()
    ns = dslash_ns(lat, b32)
    res["next2_f32_dslash"] = {"ns_per_site": ns, "gbs_algorithmic": DSLASH_BYTES[18] / 2 / ns,
                               "gbs_dram_model": DSLASH_DRAM_MODEL[18] / 2 / ns}
    x32 = lat.new_vector(len(shifts), dtype=torch.float32)
    s_it, n = cg_s_per_iter(lat, lambda: lat.mshift_cg(b32, shifts, tol, x=x32, raise_on_noconv=False)[1])
    res["next2_f32_mshift_cg"] = {"s_per_iter": s_it, "iters": n,
                                  "note": "float links, vectors and sweeps; scalar products and recurrences in double"}
    lat.close()
    # NEXT-2, mixed precision: full solves to tol on the true residual, against the double-precision solver
    lat = lq.Lattice(L, mass=mass, precisions=lq.LQCD_PREC_F64 | lq.LQCD_PREC_F32)
    lat.set_gauge(U)
    lat.set_option(lq.LQCD_OPT_MAX_ITER, 100000)
    mixed = {}
    for name, sh in (("one_system", shifts[:1]), ("all_systems", shifts)):
        xm = lat.new_vector(len(sh))
        _, im = lat.mshift_cg_mixed(b, sh, tol, x=xm, raise_on_noconv=False)
        _, idb = lat.mshift_cg(b, sh, tol, x=xm, raise_on_noconv=False)
        mixed[name] = {"nshift": len(sh), "mixed_s": im["solve_ms"] * 1e-3, "mixed_float_iters": im["iters"],
                       "reliable_updates": im["reliable_updates"], "mixed_true_rel_res": im["rel_res"],
                       "double_s": idb["solve_ms"] * 1e-3, "double_iters": idb["iters"]}
        del xm
    mixed["note"] = ("lqcd_mshift_cg_mixed (float CG + double reliable updates; with several systems a float "
                     "multi-shift phase, then each system finished alone) against lqcd_mshift_cg, solves to convergence")
    res["next2_mixed"] = mixed
    lat.close()
    return res


def n_active_schedule(freeze_iter, iters):
    """number of shifts updated in iteration j = 1..iters (shift i is updated while j <= freeze_iter[i])"""
    return [sum(1 for fz in freeze_iter if j <= fz) for j in range(1, iters + 1)]


def run_ours(args, world, rank, local):
    import paper_1801_01473_b200 as lq
    lq.load_library()
    assert torch.cuda.is_available(), "bench.py needs a GPU for --impl ours (there is no CPU fallback)"
    torch.cuda.set_device(local)
    cfg = gen.CONFIGS[args.workload]
    L, mass, shifts, tol = cfg["L"], cfg["mass"], cfg["shifts"], cfg["tol"]
    K, W = args.steps, args.warmup
    recon = args.recon
    peak, peak_src = load_peaks()
    stream = torch.cuda.Stream()
    out = {}
    slab = args.parallel == "slab"
    Lg = tuple(L[:3]) + (L[3] * world,)                 # slab mode: weak scaling, the lattice grows along t
    with torch.cuda.stream(stream):
        if slab:
            U = gen.random_su3_links_slab(Lg, rank, world, device="cuda")
            f = gen.gaussian_field_slab(Lg, rank, world, device="cuda")
            lat = lq.Lattice(Lg, mass=mass, recon=recon, slab=(rank, world), comm="nccl")
        else:
            U = gen.random_su3_links(L, device="cuda")
            f = gen.gaussian_field(L, device="cuda")
            lat = lq.Lattice(L, mass=mass, recon=recon)
        lat.set_gauge(U)
        b = lat.pack(f, 0)
        x = lat.new_vector(len(shifts))

        phase('inputs drawn, gauge stored')
        # ---- warm-up: W iterations (also builds the CUDA graph)
        lat.set_option(lq.LQCD_OPT_MAX_ITER, max(W, 3))
        lat.mshift_cg(b, shifts, tol, x=x, raise_on_noconv=False)

        # ---- timed: exactly K iterations, barrier + synchronize on both sides, clocks sampled meanwhile
        lat.set_option(lq.LQCD_OPT_MAX_ITER, K)
        torch.cuda.synchronize()
        barrier(world)
        n0 = lat.launches
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(local) as clocks:
            e0.record()
            _, info = lat.mshift_cg(b, shifts, tol, x=x, raise_on_noconv=False)
            e1.record()
            torch.cuda.synchronize()
        barrier(world)
        assert info["iters"] == K, f"solver stopped after {info['iters']} < K={K} iterations; lower --steps"
        ms_total, _, _ = aggregate_replicas(world, e0.elapsed_time(e1), K)
        launches = lat.launches - n0
        sched = n_active_schedule(info["freeze_iter"], K)
        bytes_total = sum(cg_bytes_per_site(n, recon) for n in sched) * lat.Vh
        m_blk = int(lat.get_option(lq.LQCD_OPT_SHIFT_BLOCK))
        bytes_moved = cg_bytes_moved(info["freeze_iter"], K, m_blk, recon) * lat.Vh
        out["timed"] = dict(ms_total=ms_total, launches=launches, launches_all=int(sum_over_ranks(world, launches)),
                            n_active_mean=sum(sched) / K, shift_block=m_blk,
                            gbs_algorithmic=bytes_total / (ms_total * 1e6),
                            gbs_moved=bytes_moved / (ms_total * 1e6), kernel_ms=info["solve_ms"])

        phase('timed region done')
        # ---- e2e: same K iterations through the host-pointer entry point (rank-local, then max)
        b_host = torch.empty(b.shape, dtype=torch.float64, pin_memory=True)
        b_host.copy_(b)
        x_host = torch.empty(x.shape, dtype=torch.float64, pin_memory=True)
        lat.set_option(lq.LQCD_OPT_MAX_ITER, max(W, 3))
        lat.mshift_cg(b_host, shifts, tol, x=x_host, raise_on_noconv=False)
        lat.set_option(lq.LQCD_OPT_MAX_ITER, K)
        torch.cuda.synchronize()
        barrier(world)
        t0 = time.perf_counter()
        e0.record()
        _, info_h = lat.mshift_cg(b_host, shifts, tol, x=x_host, raise_on_noconv=False)
        e1.record()
        torch.cuda.synchronize()
        wall_ms = (time.perf_counter() - t0) * 1e3
        e2e_ms = max_over_ranks(world, max(e0.elapsed_time(e1), wall_ms))
        assert info_h["iters"] == K
        assert torch.equal(x_host, x.cpu()), "host entry point and device entry point disagree"
        out["e2e"] = dict(ms_total=e2e_ms, h2d=b_host.numel() * 8, d2h=x_host.numel() * 8)
        del b_host, x_host

        phase('e2e done')
        if (rank == 0 or slab) and not args.quick:
            # ---- the same solve to convergence (what a user runs): average s/iter, iteration count
            lat.set_option(lq.LQCD_OPT_MAX_ITER, 100000)
            _, full = lat.mshift_cg(b, shifts, tol, x=x, raise_on_noconv=False)
            sched_f = n_active_schedule(full["freeze_iter"], full["iters"])
            bytes_f = sum(cg_bytes_per_site(n, recon) for n in sched_f) * lat.Vh
            moved_f = cg_bytes_moved(full["freeze_iter"], full["iters"], m_blk, recon) * lat.Vh
            out["full_solve"] = dict(iters=full["iters"], status=full["status"], rel_res=full["rel_res"],
                                     s_per_iter=full["solve_ms"] * 1e-3 / max(full["iters"], 1),
                                     solve_s=full["solve_ms"] * 1e-3, n_active_mean=sum(sched_f) / max(len(sched_f), 1),
                                     gbs_algorithmic=bytes_f / (full["solve_ms"] * 1e6),
                                     gbs_moved=moved_f / (full["solve_ms"] * 1e6),
                                     freeze_iter=full["freeze_iter"])
        lat.close()

        if rank == 0 and not args.quick and not slab:
            # ---- the same K iterations with the other link format (BASELINE config 3 compares the two; the paper
            # always runs with two-row links)
            other = 12 if recon == 18 else 18
            lat2 = lq.Lattice(L, mass=mass, recon=other)
            lat2.set_gauge(U)
            lat2.set_option(lq.LQCD_OPT_MAX_ITER, max(W, 3))
            lat2.mshift_cg(b, shifts, tol, x=x, raise_on_noconv=False)
            lat2.set_option(lq.LQCD_OPT_MAX_ITER, K)
            _, info2 = lat2.mshift_cg(b, shifts, tol, x=x, raise_on_noconv=False)
            out[f"cg_recon{other}"] = dict(s_per_iter=info2["solve_ms"] * 1e-3 / max(info2["iters"], 1), iters=info2["iters"],
                                           note=f"same {K} iterations with {other}-real links, device time of the solve")
            lat2.close()
        del x

        phase('full solve / other link format done')
        # ---- the dominant kernel alone: D_oe / D_eo at the workload size, live CUDA events
        reps = max(K // 2, 20)
        ds = {}
        if rank == 0:
            name = "x".join(str(v) for v in L)
            ds[name] = {f"recon{recon}": time_dslash(lq, L, recon, reps, 5, U, f)}
            if not args.quick:
                other = 12 if recon == 18 else 18
                ds[name][f"recon{other}"] = time_dslash(lq, L, other, reps, 5, U, f)
        if slab:
            out["dslash_slab"] = time_dslash(lq, L, recon, reps, 5, U, f, slab=(Lg, rank, world))
        phase('dslash at workload size done')
        if rank == 0 and not args.quick and not slab:
            out["next_rows"] = time_next_rows(lq, L, mass, shifts, tol, K, W, U, f)
            out["read_only_gbs"] = read_only_reference_gbs()
        del U, f
        phase('next rows done')
        if rank == 0 and not args.quick and args.workload == "config4_48^4":
            L3 = gen.CONFIGS["config3_32^4"]["L"]
            U3, f3 = gen.random_su3_links(L3, device="cuda"), gen.gaussian_field(L3, device="cuda")
            ds["32x32x32x32"] = {f"recon{r}": time_dslash(lq, L3, r, 500, 20, U3, f3) for r in (18, 12)}
            del U3, f3
        out["dslash"] = ds
    out["clocks"] = clocks.summary()
    out["peak"] = (peak, peak_src)
    out["cfg"] = dict(L=L, mass=mass, nshift=len(shifts), tol=tol, recon=recon)
    return out


# ---------------------------------------------------------------------------------------------------
# the CPU oracle (cpu_baseline leg, and the whole of --impl reference)
# ---------------------------------------------------------------------------------------------------
def run_oracle(workload: str, budget_s: float, steps: int | None, warmup: int = 0):
    """Times the oracle's multi-shift CG on the workload's inputs.  Returns (s_per_iter, description).
    Without `steps`, the number of iterations is chosen so that the run takes about budget_s."""
    import oracle
    cfg = gen.CONFIGS[workload]
    L, mass, shifts, tol = cfg["L"], cfg["mass"], cfg["shifts"], cfg["tol"]
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    U = gen.random_su3_links(L, device=dev).cpu().numpy()
    f = gen.gaussian_field(L, device=dev).cpu().numpy()
    b = oracle.restrict(L, 0, f)
    del f
    cores = oracle.num_threads()
    oracle.mshift_cg(L, U, mass, b, shifts, tol, max_iter=1)          # first touch of the work arrays
    t0 = time.perf_counter()
    oracle.mshift_cg(L, U, mass, b, shifts, tol, max_iter=2)
    t1 = (time.perf_counter() - t0) / 2
    if steps is None:
        steps = int(max(2, min(200, budget_s / max(t1, 1e-3))))
    else:
        # keep the whole reference run within a few minutes: cap the iterations actually executed
        cap = int(max(2, budget_s / max(t1, 1e-3)))
        steps = min(steps, cap)
    for _ in range(min(warmup, 1)):
        oracle.mshift_cg(L, U, mass, b, shifts, tol, max_iter=1)
    t0 = time.perf_counter()
    _, info = oracle.mshift_cg(L, U, mass, b, shifts, tol, max_iter=steps)
    dt = time.perf_counter() - t0
    sample = (f"{info['iters']} CG iterations of {workload} ({len(shifts)} shifts, all active) incl. solver set-up, "
              f"OpenMP on {cores} threads, {dt:.1f} s")
    return dt / info["iters"], cores, sample, info["iters"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config4_48^4", choices=sorted(gen.CONFIGS))
    ap.add_argument("--recon", type=int, default=18, choices=[18, 12])
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default; north_star: no sharding) or ONE lattice of N times "
                         "the time extent cut into N slabs (NEXT-3; faces over NCCL, all-reduced scalar products). "
                         "With N = 1, slab runs the slab code path on one rank (ring closed on itself).")
    ap.add_argument("--next-rows-only", action="store_true",
                    help="run only the widened rows (rational sum, f32, U(1) phases) and print their JSON object "
                         "(used for the ncu captures of those kernels)")
    ap.add_argument("--quick", action="store_true", help="skip the full solve, the 32^4 table and the CPU baseline")
    ap.add_argument("--cpu-budget", type=float, default=20.0, help="seconds of oracle time for cpu_baseline")
    args = ap.parse_args()
    if args.next_rows_only:
        import paper_1801_01473_b200 as lq
        cfg = gen.CONFIGS[args.workload]
        with torch.cuda.stream(torch.cuda.Stream()):
            U = gen.random_su3_links(cfg["L"], device="cuda")
            f = gen.gaussian_field(cfg["L"], device="cuda")
            res = time_next_rows(lq, cfg["L"], cfg["mass"], cfg["shifts"], cfg["tol"], args.steps, args.warmup, U, f)
        print(json.dumps({"next_rows": res}))
        return 0
    if args.impl == "reference" and int(os.environ.get("RANK", "0")) != 0:
        return 0                                   # the oracle arm runs on rank 0 alone, no process group
    if args.impl == "reference":
        world, rank, local = 1, 0, 0
    else:
        world, rank, local = dist_setup(args.gpus)
    cfg = gen.CONFIGS[args.workload]
    lname = "x".join(str(v) for v in cfg["L"])
    config = {"workload": f"{args.workload}: {lname} lattice, multi-shift CG with {len(cfg['shifts'])} shifts "
                          f"(geometric {cfg['shifts'][0]:g}..{cfg['shifts'][-1]:g}), m={cfg['mass']}, tol={cfg['tol']:g}, "
                          f"{args.recon}-real links, seeded random SU(3) links + Gaussian even-site source",
              "step": "one multi-shift CG iteration (D_oe, D_eo+epilogue, scalar recurrences, r update, base x/p update, "
                      "1/m of the block sweep over the shifted x_i/p_i)",
              "lattice": list(cfg["L"]), "nshift": len(cfg["shifts"]), "mass": cfg["mass"], "tol": cfg["tol"],
              "recon": args.recon,
              "parallelism": (f"1-D slabs along t: ONE {lname[:lname.rfind('x')]}x{cfg['L'][3] * world} lattice over {world} "
                              f"rank(s), value = s/iter of that solve / {world}") if args.parallel == "slab"
              else ("replicas only" if world > 1 else "single GPU"),
              "l2": "inputs larger than L2 (links 3.06 GB vs 126 MB); no flush needed"}

    if args.impl == "reference":
        s_iter, cores, sample, n = run_oracle(args.workload, budget_s=150.0, steps=args.steps, warmup=args.warmup)
        line = {"impl": "reference", "metric": "mshift_cg_s_per_iter", "value": s_iter, "unit": "s/iter",
                "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": s_iter * 1e3,
                "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic", "config": config,
                "cpu_baseline": {"value": s_iter, "unit": "s/iter", "cores": cores, "kind": "oracle", "sample": sample},
                "e2e": {"value": s_iter, "unit": "s/iter", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "steps_executed": n}
        print(json.dumps(line))
        return 0

    res = run_ours(args, world, rank, local)
    if rank != 0:
        barrier(world)
        return 0
    K, W = args.steps, args.warmup
    peak, peak_src = res["peak"]
    ms_step = res["timed"]["ms_total"] / K
    value = ms_step * 1e-3 / world                     # replicas: N solves advance one iteration per ms_step
    ds_main = res["dslash"][lname][f"recon{args.recon}"]
    bytes_per_launch = ds_main["bytes_per_launch"]
    achieved = ds_main["gbs_algorithmic"]
    traffic = NCU_DRAM_BYTES_PER_LAUNCH.get((args.workload, args.recon))
    line = {
        "metric": "mshift_cg_s_per_iter", "value": value, "unit": "s/iter", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": config,
        "clocks": res["clocks"],
        "e2e": {"value": res["e2e"]["ms_total"] * 1e-3 / K / world, "unit": "s/iter",
                "h2d_bytes_per_step": res["e2e"]["h2d"] / K, "d2h_bytes_per_step": res["e2e"]["d2h"] / K,
                "note": "lqcd_mshift_cg_host: pinned-host b in, 16 pinned-host solutions out, K iterations per call"},
        "gpu_launches": res["timed"]["launches_all"],
        "roofline": {"bound": "hbm", "kernel": f"dslash_kernel<{args.recon},0|1> (D_oe / D_eo) at {lname}",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "peak_source": peak_src,
                     "bytes_per_launch": bytes_per_launch, "us_per_launch": ds_main["us_per_application"],
                     "ns_per_site": ds_main["ns_per_site"],
                     "achieved_dram_model": ds_main["gbs_dram_model"], "frac_dram_model": ds_main["gbs_dram_model"] / peak,
                     "frac_of_nominal_8000": achieved / 8000.0,
                     "read_only_reference_gbs": res.get("read_only_gbs"),
                     "note": "achieved = algorithmic bytes (8 links + 8 neighbour vectors + 1 output per site) / event "
                             "time; the 8 neighbour-vector reads are mostly L2 hits, achieved_dram_model counts each "
                             "input vector once (what DRAM must deliver)"},
        "cg": {"n_active_mean": res["timed"]["n_active_mean"], "shift_block": res["timed"]["shift_block"],
               "gbs_algorithmic": res["timed"]["gbs_algorithmic"], "gbs_moved": res["timed"]["gbs_moved"],
               "frac_of_peak_moved": res["timed"]["gbs_moved"] / peak,
               "note": "gbs_algorithmic: bytes of the per-iteration method (SURVEY.md 8(d): 3600+192(n_act-1) B/site) / time, "
                       "an equivalent rate; gbs_moved: bytes the block-deferred updates actually move / time"},
        "dslash": res["dslash"],
    }
    if "full_solve" in res:
        line["full_solve"] = res["full_solve"]
    if "dslash_slab" in res:
        line["dslash_slab"] = res["dslash_slab"]
    for key in ("cg_recon12", "cg_recon18", "next_rows"):
        if key in res:
            line[key] = res[key]
    phase("GPU part done")
    if not args.quick and world == 1:
        s_iter, cores, sample, _ = run_oracle(args.workload, budget_s=args.cpu_budget, steps=None)
        line["cpu_baseline"] = {"value": s_iter, "unit": "s/iter", "cores": cores, "kind": "oracle", "sample": sample}
    phase("CPU baseline done")
    print(json.dumps(line))
    barrier(world)
    return 0


if __name__ == "__main__":
    sys.exit(main())
