#!/usr/bin/env python
"""bench.py -- the BASELINE.json metric on one B200 (or on N GPUs of one node).

Metric (BASELINE.json): "Dslash ns/site and HBM GB/s (fraction of peak), 1xB200 double; mshift-CG s/iter".

  step      one iteration of the multi-shift CG = one pass of the whole hot path (DESIGN.md rows A2-A9:
            D_oe, D_eo with every sum and scalar product fused into the two operator sweeps, scalar recurrences,
            1/m of the block sweep over the x_i/p_i of the active shifts, loop control); A1 (link storage) is
            one-time set-up.
  workload  BASELINE config 4: 48^4, 16 shifts geometric 1e-5..1, m = 0.0075, tol 1e-10, 18-real links,
            seeded random SU(3) links + Gaussian even-site source (lqcd_inputs).  Links (3.06 GB) are far
            larger than L2, so no explicit L2 flush is needed between iterations.
  value     seconds per CG iteration over exactly K iterations (device time, CUDA events), inputs resident in
            HBM; `value_steady` is the same over 96 iterations (a whole number of shift blocks).
  roofline  the D_oe/D_eo kernel alone at 48^4 (18-real): DRAM-compulsory bytes (every link, every
            input vector and the output once = 1248 B/site) / live CUDA-event time, against the measured HBM
            copy bandwidth; the algorithmic rate (1584 B/site, neighbour re-reads served by L1/L2) beside it.
  cg_roofline  the same for the timed CG iterations, bytes from the recorded freeze schedule.
  dslash    ns/site and GB/s of the operator alone at 32^4 and 48^4, 18- and 12-real links.
  small     BASELINE config 2 (16^4, whole solve) and the same shifts at 32^4: s/iter, against an L2 read stream.
  e2e       the same K iterations through lqcd_mshift_cg_host: b from pinned host memory, all 16 solutions back to
            pinned host memory, copies inside the timed region; `e2e_rational`: lqcd_rational_apply_host (what the
            RHMC calls: one vector in, one vector back).
  cpu_baseline  the CPU oracle (oracle/, as it stands) on the host cores: CG s/iter on a few iterations of the
            same workload, Dslash ns/site at 32^4 (all cores and 1 thread), the whole 16^4 solve.
            `--impl reference` runs only the CG part.

N > 1: `python bench.py --gpus N` starts its own N ranks (torch.distributed.run) unless it already runs under
torchrun.  Replicas are the headline (north_star: no sharding); rank 0 then runs the 1-D slab path (NEXT-3) on all N
GPUs as a guarded sub-run and reports it under `slab`.

Usage:  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]
"""
from __future__ import annotations

import argparse
import json
import os
import signal
import socket
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

import lqcd_inputs as gen  # noqa: E402

# Bytes per output site of one parity application.
LINK_BYTES = {18: 144, 12: 96}
DSLASH_BYTES = {r: 8 * LINK_BYTES[r] + 8 * 48 + 48 for r in (18, 12)}            # algorithmic: 1584 / 1200
DSLASH_DRAM_MODEL = {r: 8 * LINK_BYTES[r] + 48 + 48 for r in (18, 12)}          # DRAM-compulsory: 1248 / 864
DSLASH_FLOPS = {18: 570, 12: 570 + 8 * 42}

# DRAM bytes per launch of the plain D_oe/D_eo kernel measured by `ncu --set full` (dram__bytes_read.sum +
# dram__bytes_write.sum), keyed by (workload, recon): (read GB, write GB, file under profiles/ that holds them).
# tests/test_host_logic.py checks these constants against that file.
NCU_DRAM_GB_PER_LAUNCH = {
    ("config4_48^4", 18): (3.190677, 0.104111, "profiles/ncu_full_r02.md"),
    ("config4_48^4", 12): (2.171204, 0.101689, "profiles/ncu_full_r01.md"),
}


def cg_bytes_per_site(n_active: int, recon: int) -> int:
    """SURVEY.md §8(d) model of one CG iteration per even site of the METHOD as the paper states it (shift updates
    applied every iteration, one sweep per BLAS-1 operation): two Dslash + p in the epilogue + r update + base x/p
    + 192 B per further active shift.  An equivalent rate only: the library moves fewer bytes (cg_dram_bytes)."""
    return 2 * DSLASH_BYTES[recon] + 48 + 144 + 240 + 192 * (n_active - 1)


def cg_dram_bytes(freeze_iter, iters: int, m: int, recon: int) -> int:
    """DRAM-compulsory bytes per even site of `iters` iterations as the library runs them:
      K1  8 links + r + p_old in, t out;   K2  8 links + t + r + p_old in, p + r_new out;
      m >= 2: per block of m iterations p_keep out (48), and one sweep: the block's residuals in (48 each), x_i, p_i
              in and out (192) of every shifted system active when the block began, p_keep in + x_0 in/out (144);
      m == 1: x_0 in/out in K2 (96); per iteration the residual (48) + 192 per active shifted system;
      the last sweep of a solve does not write the p_i (48 per shifted system less)."""
    links = 8 * LINK_BYTES[recon]
    base = max(range(len(freeze_iter)), key=lambda i: freeze_iter[i])
    total = iters * (2 * links + 3 * 48 + 5 * 48)
    for n0 in range(0, iters, m):
        nres = min(m, iters - n0)
        n_in = sum(1 for i, fz in enumerate(freeze_iter) if i != base and fz > n0)
        if m >= 2 and n0 == 0:
            # first sweep of a solve: P = b read once for all shifted systems, X = 0 not read (cg.cuh, first_block)
            total += 48 + 48 * nres + 48 + 96 * n_in + 96
        elif m >= 2:
            total += 48 + 48 * nres + 192 * n_in + 144
        else:
            total += 96 + (48 + 192 * n_in if n_in else 0)
        if n0 + m >= iters:
            total -= 48 * n_in      # the sweep that ends the solve does not store the p_i (nothing reads them any more)
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
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs: copy, read+write bytes, best of 10)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU while the timed region runs (pynvml thread)."""

    def __init__(self, index: int, period: float = 0.002):
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._warm = threading.Event()      # set once the first (discarded) poll is through: NVML's first call is slow
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
        try:
            nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
        except Exception:
            pass
        self._warm.set()
        self._armed.wait()
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
        """Starts the polling thread and returns once it is ready; samples are taken from arm() on."""
        self._armed = threading.Event()
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
            self._warm.wait(2.0)
        return self

    def arm(self):
        self._armed.set()

    def __exit__(self, *exc):
        self._stop.set()
        self._armed.set()
        if self._thread is not None:
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------------
# ranks
# ---------------------------------------------------------------------------------------------------
def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def torchrun_cmd(n: int, script_args: list[str]) -> list[str]:
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
            "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + script_args


def self_launch(args, argv: list[str]):
    """`python bench.py --gpus N` with N > 1 outside torchrun: become N ranks.  Never runs fewer GPUs than asked."""
    if args.gpus <= 1 or "WORLD_SIZE" in os.environ or args.impl == "reference":
        return
    if not args.plumbing_check:
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            print(f"bench.py: --gpus {args.gpus} needs {args.gpus} CUDA devices, this machine has {have}",
                  file=sys.stderr)
            sys.exit(2)
    cmd = torchrun_cmd(args.gpus, argv)
    os.execv(sys.executable, cmd)


def dist_setup(n_gpus: int):
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != max(n_gpus, 1):
        print(f"bench.py: --gpus {n_gpus} but WORLD_SIZE={world}", file=sys.stderr)
        sys.exit(2)
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        if torch.cuda.is_available():
            torch.cuda.set_device(local)
        dist.init_process_group(backend=backend)
    return world, rank, local


def dist_teardown(world):
    if world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()


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
    time the job advanced world*steps iterations.  Returns (ms_total, ms_per_step of one replica, aggregate s/iter)."""
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


def run_plumbing_check(args):
    """The multi-rank plumbing of this file without a GPU or the library (gloo on the CPU box): launch, process
    group, barriers, max / sum over ranks, the replica normalisation.  tests/test_bench_dist.py runs it."""
    world, rank, local = dist_setup(args.gpus)
    barrier(world)
    ms_total, ms_step, value = aggregate_replicas(world, 10.0 * (rank + 1), args.steps)
    launches = sum_over_ranks(world, 100 + rank)
    barrier(world)
    if rank == 0:
        print(json.dumps({"plumbing_check": True, "n_gpus": world, "steps": args.steps, "ms_total": ms_total,
                          "ms_per_step": ms_step, "value": value, "launches": launches}))
    dist_teardown(world)
    return 0


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def ev():
    return torch.cuda.Event(enable_timing=True)


def time_dslash(lq, L, recon, reps, warm, links=None, field=None, slab=None, comm="nccl", u1=False):
    """ns/site and GB/s of one parity application: reps x (D_oe: b->t, D_eo: t->u) with fixed b
    (never fed back: |D| ~ 2.6 on random links would overflow).  slab = (L_global, rank, nranks): the same on a slab
    context (two face exchanges over NCCL, interior and border launches per application); collective.
    u1: with a general U(1) phase per link (8 angles of 8 bytes per site more to read)."""
    U = links if links is not None else gen.random_su3_links(L, device="cuda")
    f = field if field is not None else gen.gaussian_field(L, device="cuda")
    lat = lq.Lattice(L, recon=recon) if slab is None else lq.Lattice(slab[0], recon=recon, slab=slab[1:], comm=comm)
    lat.set_gauge(U)
    if u1:
        lat.set_u1_phases(gen.random_u1_phases(L, device="cuda"))
    b = lat.pack(f, 0)
    t = torch.empty_like(b)
    u = torch.empty_like(b)
    for _ in range(warm):
        lat.doe(b, out=t)
        lat.deo(t, out=u)
    e0, e1 = ev(), ev()
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
    extra = 64 if u1 else 0                  # 8 angles x 8 bytes per site
    return {"us_per_application": ms * 1e3, "ns_per_site": ns_site,
            "gbs_dram_model": (DSLASH_DRAM_MODEL[recon] + extra) / ns_site,
            "gbs_algorithmic": (DSLASH_BYTES[recon] + extra) / ns_site,
            "gflops": DSLASH_FLOPS[recon] / ns_site, "launches": launches,
            "dram_bytes_per_launch": (DSLASH_DRAM_MODEL[recon] + extra) * lat.Vh,
            "algorithmic_bytes_per_launch": (DSLASH_BYTES[recon] + extra) * lat.Vh}


def read_stream_gbs(nbytes: int, reps: int = 10):
    """What a plain read-only stream reaches on this GPU over a buffer of nbytes (torch.sum over doubles, best of
    `reps` after 3 warm-up passes, CUDA events).  4 GiB: HBM (the measured peak of MEASURED_PEAKS.json is a COPY, half
    writes; the Dslash is 97 % reads).  40 MB: the buffer stays in L2 (126 MB), i.e. an L2 read stream."""
    a = torch.ones(nbytes // 8, dtype=torch.float64, device="cuda")
    best = 0.0
    for i in range(reps + 3):
        e0, e1 = ev(), ev()
        e0.record()
        a.sum()
        e1.record()
        torch.cuda.current_stream().synchronize()
        if i >= 3:
            best = max(best, a.numel() * 8 / (e0.elapsed_time(e1) * 1e6))
    del a
    return best


def time_small(lq, peak):
    """The small-lattice regime (SURVEY.md §7 "Small lattices are launch-bound", BASELINE config 2): the whole 16^4
    solve, and the same 8 shifts at 32^4 (400 iterations, then the whole solve).  At 16^4 the links (37.7 MB) and
    part of the vectors are served by L2, so the rate is quoted against an L2 read stream measured here, not against
    HBM.  `driver` says which of the two drivers of the iteration the library chose."""
    cfg = gen.CONFIGS["config2_16^4"]
    out = {}
    for name, L in (("16x16x16x16", cfg["L"]), ("32x32x32x32", (32, 32, 32, 32))):
        U, f = gen.random_su3_links(L, device="cuda"), gen.gaussian_field(L, device="cuda")
        lat = lq.Lattice(L, mass=cfg["mass"])
        lat.set_gauge(U)
        b = lat.pack(f, 0)
        x = lat.new_vector(len(cfg["shifts"]))
        m = int(lat.get_option(lq.LQCD_OPT_SHIFT_BLOCK))
        lat.set_option(lq.LQCD_OPT_MAX_ITER, 32)
        lat.mshift_cg(b, cfg["shifts"], cfg["tol"], x=x, raise_on_noconv=False)
        lat.set_option(lq.LQCD_OPT_MAX_ITER, 400)
        _, first = lat.mshift_cg(b, cfg["shifts"], cfg["tol"], x=x, raise_on_noconv=False)
        lat.set_option(lq.LQCD_OPT_MAX_ITER, 100000)
        n0 = lat.launches
        _, full = lat.mshift_cg(b, cfg["shifts"], cfg["tol"], x=x, raise_on_noconv=False)
        n_launch = lat.launches - n0
        moved = cg_dram_bytes(full["freeze_iter"], full["iters"], m, 18) * lat.Vh
        gbs = moved / (full["solve_ms"] * 1e6)
        out[name] = {"iters": full["iters"], "status": full["status"], "rel_res": full["rel_res"],
                     "s_per_iter": full["solve_ms"] * 1e-3 / max(full["iters"], 1),
                     "s_per_iter_first_400": first["solve_ms"] * 1e-3 / max(first["iters"], 1),
                     "solve_s": full["solve_ms"] * 1e-3, "freeze_iter": full["freeze_iter"],
                     "gbs_moved": gbs, "gbs_moved_over_hbm_peak": gbs / peak,
                     "served_from": ("L2 for the most part (links + vectors fit): gbs_moved is NOT a DRAM rate"
                                     if 8 * 9 * lat.Vh * 16 <= (48 << 20) else "DRAM"),
                     "launches_per_iter": n_launch / max(full["iters"], 1),
                     "driver": ("CUDA graph of the iteration's launches" if full.get("graph_replays") else
                                "one persistent cooperative kernel" if n_launch < 8 else "plain launches")}
        lat.close()
        del U, f, x, b
    out["note"] = ("config 2 (16^4, m=0.01, 8 shifts, tol 1e-10) whole solve, and the same at 32^4; gbs_moved = ALGORITHMIC "
                   "bytes the iteration touches (cg_dram_bytes) / time.  At 16^4 they come out of L2, so gbs_moved over the "
                   "HBM peak is a ratio of two different things, not a roofline fraction; no L2 ceiling is quoted: a one-"
                   "stream L2 read microbenchmark gave 2.2 TB/s, which the solver exceeds 2.3x, so it is not a ceiling.  The "
                   "yardstick for small lattices is time: two bare operator applications from L2 are 9 us at 16^4")
    return out


def time_next_rows(lq, L, mass, shifts, tol, K, W, U, f):
    """The widened rows on the same workload, K iterations / applications each, device time:
    NEXT-1 rational sum, NEXT-2 single precision (Dslash and CG), NEXT-4 general U(1) phases (Dslash)."""
    res = {}

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
            lat = lq.Lattice(Lg, mass=mass, recon=recon, slab=(rank, world), comm=args.slab_comm)
        else:
            U = gen.random_su3_links(L, device="cuda")
            f = gen.gaussian_field(L, device="cuda")
            lat = lq.Lattice(L, mass=mass, recon=recon)
        lat.set_gauge(U)
        b = lat.pack(f, 0)
        x = lat.new_vector(len(shifts))
        m_blk = int(lat.get_option(lq.LQCD_OPT_SHIFT_BLOCK))

        phase('inputs drawn, gauge stored')
        # ---- warm-up: W iterations (also builds the CUDA graph)
        lat.set_option(lq.LQCD_OPT_MAX_ITER, max(W, 3))
        lat.mshift_cg(b, shifts, tol, x=x, raise_on_noconv=False)

        # ---- timed: exactly K iterations, barrier + synchronize on both sides, clocks sampled meanwhile
        lat.set_option(lq.LQCD_OPT_MAX_ITER, K)
        torch.cuda.synchronize()
        barrier(world)
        n0 = lat.launches
        e0, e1 = ev(), ev()
        with ClockSampler(local) as clocks:
            clocks.arm()
            e0.record()
            _, info = lat.mshift_cg(b, shifts, tol, x=x, raise_on_noconv=False)
            e1.record()
            torch.cuda.synchronize()
        barrier(world)
        assert info["iters"] == K, f"solver stopped after {info['iters']} < K={K} iterations; lower --steps"
        ms_total, _, _ = aggregate_replicas(world, e0.elapsed_time(e1), K)
        launches = lat.launches - n0
        sched = n_active_schedule(info["freeze_iter"], K)
        bytes_method = sum(cg_bytes_per_site(n, recon) for n in sched) * lat.Vh
        bytes_dram = cg_dram_bytes(info["freeze_iter"], K, m_blk, recon) * lat.Vh
        out["timed"] = dict(ms_total=ms_total, launches=launches, launches_all=int(sum_over_ranks(world, launches)),
                            n_active_mean=sum(sched) / K, shift_block=m_blk, bytes_dram=bytes_dram,
                            gbs_method_equivalent=bytes_method / (ms_total * 1e6),
                            gbs_dram=bytes_dram / (ms_total * 1e6), kernel_ms=info["solve_ms"])

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
        del x_host
        # what the RHMC calls: the rational function applied to a host vector, one vector back
        if not slab:
            alpha = [1.0 / (1 + i) for i in range(len(shifts))]
            y_host = torch.empty(b.shape, dtype=torch.float64, pin_memory=True)
            lat.set_option(lq.LQCD_OPT_MAX_ITER, max(W, 3))
            lat.rational_apply(b_host, 0.5, alpha, shifts, tol, y=y_host, raise_on_noconv=False)
            lat.set_option(lq.LQCD_OPT_MAX_ITER, K)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            e0.record()
            _, info_r = lat.rational_apply(b_host, 0.5, alpha, shifts, tol, y=y_host, raise_on_noconv=False)
            e1.record()
            torch.cuda.synchronize()
            wall_ms = (time.perf_counter() - t0) * 1e3
            out["e2e_rational"] = dict(ms_total=max(e0.elapsed_time(e1), wall_ms), iters=info_r["iters"],
                                       h2d=b_host.numel() * 8, d2h=y_host.numel() * 8, kernel_ms=info_r["solve_ms"])
            del y_host
        del b_host

        phase('e2e done')
        if rank == 0 or slab:
            # ---- the same over a whole number of shift blocks (the driver's K need not be one)
            Ks = 96
            lat.set_option(lq.LQCD_OPT_MAX_ITER, Ks)
            _, st = lat.mshift_cg(b, shifts, tol, x=x, raise_on_noconv=False)
            out["steady"] = dict(iters=st["iters"], s_per_iter=st["solve_ms"] * 1e-3 / max(st["iters"], 1),
                                 gbs_dram=cg_dram_bytes(st["freeze_iter"], st["iters"], m_blk, recon) * lat.Vh
                                 / (st["solve_ms"] * 1e6))
        if (rank == 0 or slab) and not args.quick:
            # ---- the same solve to convergence (what a user runs): average s/iter, iteration count
            lat.set_option(lq.LQCD_OPT_MAX_ITER, 100000)
            _, full = lat.mshift_cg(b, shifts, tol, x=x, raise_on_noconv=False)
            sched_f = n_active_schedule(full["freeze_iter"], full["iters"])
            bytes_f = sum(cg_bytes_per_site(n, recon) for n in sched_f) * lat.Vh
            moved_f = cg_dram_bytes(full["freeze_iter"], full["iters"], m_blk, recon) * lat.Vh
            out["full_solve"] = dict(iters=full["iters"], status=full["status"], rel_res=full["rel_res"],
                                     s_per_iter=full["solve_ms"] * 1e-3 / max(full["iters"], 1),
                                     solve_s=full["solve_ms"] * 1e-3, n_active_mean=sum(sched_f) / max(len(sched_f), 1),
                                     gbs_method_equivalent=bytes_f / (full["solve_ms"] * 1e6),
                                     gbs_dram=moved_f / (full["solve_ms"] * 1e6),
                                     frac_of_peak_dram=moved_f / (full["solve_ms"] * 1e6) / peak,
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
            lat2.set_option(lq.LQCD_OPT_MAX_ITER, max(K, 96))
            _, info2 = lat2.mshift_cg(b, shifts, tol, x=x, raise_on_noconv=False)
            out[f"cg_recon{other}"] = dict(
                s_per_iter=info2["solve_ms"] * 1e-3 / max(info2["iters"], 1), iters=info2["iters"],
                gbs_dram=cg_dram_bytes(info2["freeze_iter"], info2["iters"], m_blk, other) * lat2.Vh / (info2["solve_ms"] * 1e6),
                note=f"{info2['iters']} iterations with {other}-real links, device time of the solve")
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
            out["dslash_slab"] = time_dslash(lq, L, recon, reps, 5, U, f, slab=(Lg, rank, world), comm=args.slab_comm)
        phase('dslash at workload size done')
        if rank == 0 and not args.quick and not slab:
            out["next_rows"] = time_next_rows(lq, L, mass, shifts, tol, K, W, U, f)
            out["read_only_gbs"] = read_stream_gbs(4 << 30)
        del U, f, b
        phase('next rows done')
        if rank == 0 and not args.quick and args.workload == "config4_48^4":
            L3 = gen.CONFIGS["config3_32^4"]["L"]
            U3, f3 = gen.random_su3_links(L3, device="cuda"), gen.gaussian_field(L3, device="cuda")
            ds["32x32x32x32"] = {f"recon{r}": time_dslash(lq, L3, r, 500, 20, U3, f3) for r in (18, 12)}
            del U3, f3
            # the paper's own lattices (Fig. 4: 339 GFLOP/s, 290 GB/s per K80 board on
            # 32^3 x 48) in the paper's kernel configuration: two-row links AND U(1) phases
            for Lp in ((32, 32, 32, 48), (32, 32, 32, 64)):
                Up, fp = gen.random_su3_links(Lp, device="cuda"), gen.gaussian_field(Lp, device="cuda")
                row = {f"recon{r}": time_dslash(lq, Lp, r, 300, 20, Up, fp) for r in (18, 12)}
                row["recon12_u1"] = time_dslash(lq, Lp, 12, 300, 20, Up, fp, u1=True)
                for v in row.values():
                    v["frac_of_peak_dram_model"] = v["gbs_dram_model"] / peak
                ds["x".join(str(v) for v in Lp)] = row
                del Up, fp
            ds["note_paper_lattices"] = ("32x32x32x48 / x64 are the lattices of the paper's scaling runs; recon12_u1 (two-row "
                                         "links + theta phases, 864 + 64 compulsory B/site) is the kernel its Fig. 4 numbers "
                                         "(339 GFLOP/s, 290 GB/s per K80 board, ~4.4 ns/site) were measured on -- context, "
                                         "another machine")
            out["small"] = time_small(lq, peak)
        out["dslash"] = ds
        phase('small lattices done')
    out["clocks"] = clocks.summary()
    out["peak"] = (peak, peak_src)
    out["cfg"] = dict(L=L, mass=mass, nshift=len(shifts), tol=tol, recon=recon)
    return out


# ---------------------------------------------------------------------------------------------------
# NEXT-3 on the GPUs of this node: a guarded sub-run (a hang in a collective cannot lose the headline line)
# ---------------------------------------------------------------------------------------------------
def run_slab_check(args):
    """Runs as its own set of N ranks (`bench.py --slab-check --gpus N` under torchrun; N = 1 closes the ring on
    itself).  (1) parity on a 16^3 x 4N lattice: the gathered D_oe of the N slabs against the single-GPU kernel
    (bit for bit) and against the oracle, then 20 CG iterations against the oracle at a fixed count; (2) timing of
    ONE Lx*Ly*Lz*(Lt*N) lattice of the workload: operator us, CG s/iter, face bytes.  Prints {"slab": {...}}."""
    import numpy as np
    import oracle
    import paper_1801_01473_b200 as lq
    import torch.distributed as dist
    world, rank, local = dist_setup(args.gpus)
    torch.cuda.set_device(local)
    # what the faces and partial sums actually travelled over in THIS run.  With one rank the ring closes on the rank
    # itself: device-local copies, no link of any kind -- the figures then say what the slab machinery costs, nothing
    # about NVLink.  Neither transport has been run between two GPUs yet (include/lqcd.h, STATUS).
    res = {"n_ranks": world,
           "interconnect": ("none: one rank, ring closed on itself (device-local copies); not an NVLink measurement"
                            if world == 1 else f"{world} ranks on {min(world, torch.cuda.device_count())} GPU(s)"),
           "measured_between_gpus": bool(world > 1 and torch.cuda.device_count() >= world)}
    with torch.cuda.stream(torch.cuda.Stream()):
        # ---- (1) parity
        Lp = (16, 16, 16, 4 * world)
        mass, shifts = 0.05, [1e-3, 1e-2, 1e-1, 1.0]
        U, f = gen.random_su3_links(Lp), gen.gaussian_field(Lp)
        b_aos = oracle.restrict(Lp, 0, f.numpy())
        b_whole = torch.as_tensor(oracle.aos_to_soa(b_aos)).cuda()
        lat = lq.Lattice(Lp, mass=mass, slab=(rank, world), comm=args.slab_comm)
        lat.set_gauge(lq.Lattice.slab_of_links(U, Lp, rank, world).cuda())
        b = lq.Lattice.slab_of_vector(b_whole, Lp, rank, world)
        t = lat.doe(b)
        lat.set_option(lq.LQCD_OPT_MAX_ITER, 20)
        x, info = lat.mshift_cg(b, shifts, 1e-30, raise_on_noconv=False)
        torch.cuda.synchronize()

        def gather(v):                      # (..., 3, Vh_loc, 2) slabs -> whole-lattice vector on every rank
            if world == 1:
                return v
            parts = [torch.empty_like(v) for _ in range(world)]
            dist.all_gather(parts, v.contiguous())
            return torch.cat(parts, dim=-2)

        t_all, x_all = gather(t), gather(x)
        lat.close()
        if rank == 0:
            whole = lq.Lattice(Lp, mass=mass)
            whole.set_gauge(U.cuda())
            t_one = whole.doe(b_whole)
            whole.close()
            rel = lambda a, r: float(np.linalg.norm(a - r) / np.linalg.norm(r))
            t_ref = oracle.doe(Lp, U.numpy(), b_aos)
            x_ref, i_ref = oracle.mshift_cg(Lp, U.numpy(), mass, b_aos, shifts, 1e-30, max_iter=20)
            res["parity"] = {
                "lattice": list(Lp),
                "doe_bit_identical_to_single_gpu_kernel": bool(torch.equal(t_all, t_one)),
                "doe_rel_err_vs_oracle": rel(oracle.soa_to_aos(t_all.cpu().numpy()), t_ref),
                "cg20_max_rel_err_vs_oracle": max(rel(oracle.soa_to_aos(x_all[i].cpu().numpy()), x_ref[i])
                                                  for i in range(len(shifts))),
                "cg_iters": info["iters"], "oracle_iters": i_ref["iters"]}
            p = res["parity"]
            p["ok"] = bool(p["doe_bit_identical_to_single_gpu_kernel"] and p["doe_rel_err_vs_oracle"] <= 1e-12
                           and p["cg20_max_rel_err_vs_oracle"] <= 1e-11 and p["cg_iters"] == p["oracle_iters"] == 20)
        del U, f
        # ---- (2) timing at the workload size, weak scaling along t
        cfg = gen.CONFIGS[args.workload]
        L = cfg["L"]
        Lg = tuple(L[:3]) + (L[3] * world,)
        U = gen.random_su3_links_slab(Lg, rank, world, device="cuda")
        f = gen.gaussian_field_slab(Lg, rank, world, device="cuda")
        lat = lq.Lattice(Lg, mass=cfg["mass"], recon=args.recon, slab=(rank, world), comm=args.slab_comm)
        lat.set_gauge(U)
        b = lat.pack(f, 0)
        x = lat.new_vector(len(cfg["shifts"]))
        lat.set_option(lq.LQCD_OPT_MAX_ITER, max(args.warmup, 3))
        lat.mshift_cg(b, cfg["shifts"], cfg["tol"], x=x, raise_on_noconv=False)
        lat.set_option(lq.LQCD_OPT_MAX_ITER, args.steps)
        torch.cuda.synchronize()
        barrier(world)
        e0, e1 = ev(), ev()
        e0.record()
        _, info = lat.mshift_cg(b, cfg["shifts"], cfg["tol"], x=x, raise_on_noconv=False)
        e1.record()
        torch.cuda.synchronize()
        barrier(world)
        ms = max_over_ranks(world, e0.elapsed_time(e1))
        tt, uu = torch.empty_like(b), torch.empty_like(b)
        for _ in range(3):
            lat.doe(b, out=tt)
            lat.deo(tt, out=uu)
        torch.cuda.synchronize()
        barrier(world)
        reps = 20
        e0.record()
        for _ in range(reps):
            lat.doe(b, out=tt)
            lat.deo(tt, out=uu)
        e1.record()
        torch.cuda.synchronize()
        op_us = max_over_ranks(world, e0.elapsed_time(e1)) * 1e3 / (2 * reps)
        face = L[0] * L[1] * L[2] // 2 * 48
        res["timing"] = {"lattice": list(Lg), "iters": info["iters"], "s_per_iter": ms * 1e-3 / max(info["iters"], 1),
                         "s_per_iter_per_gpu_volume": ms * 1e-3 / max(info["iters"], 1) / world,
                         "operator_us": op_us, "face_bytes_each_way": face,
                         "face_bytes_per_application": 2 * face,
                         "transport": {"nccl": "NCCL send/recv + all-reduce",
                                       "p2p": "peer-mapped windows: faces stored into the neighbours' halo buffers, "
                                              "stream memory operations, slot all-reduce"}[args.slab_comm]}
        lat.close()
    barrier(world)
    if rank == 0:
        print(json.dumps({"slab": res}))
    dist_teardown(world)
    return 0


def guarded_slab_run(args, n: int, comm: str = "nccl", timeout_s: float = 600.0):
    """rank 0 of the headline run: start the slab check as a separate set of n ranks and wait at most timeout_s."""
    argv = ["--slab-check", "--slab-comm", comm, "--gpus", str(n), "--steps", str(args.steps), "--warmup", str(args.warmup),
            "--workload", args.workload, "--recon", str(args.recon)]
    cmd = torchrun_cmd(n, argv) if n > 1 else [sys.executable, os.path.abspath(__file__)] + argv
    env = {k: v for k, v in os.environ.items()
           if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT", "GROUP_RANK", "ROLE_RANK",
                        "LOCAL_WORLD_SIZE", "ROLE_WORLD_SIZE", "TORCHELASTIC_RUN_ID", "TORCHELASTIC_RESTART_COUNT",
                        "TORCHELASTIC_MAX_RESTARTS", "TORCHELASTIC_USE_AGENT_STORE", "TORCHELASTIC_ERROR_FILE")}
    env.setdefault("NCCL_DEBUG", "INFO")                 # NCCL's own log (rank count, transports) goes to stderr
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    t0 = time.perf_counter()
    try:
        # its own process group: a rank that hangs is killed together with its launcher
        proc = subprocess.Popen(cmd, env=env, stdout=subprocess.PIPE, stderr=sys.stderr, text=True, start_new_session=True)
        try:
            stdout, _ = proc.communicate(timeout=timeout_s)
        except subprocess.TimeoutExpired:
            os.killpg(proc.pid, signal.SIGKILL)
            proc.communicate()
            raise
        p = subprocess.CompletedProcess(cmd, proc.returncode, stdout, None)
    except subprocess.TimeoutExpired:
        return {"error": f"slab sub-run did not finish within {timeout_s:.0f} s (killed)", "n_ranks": n}
    for line in reversed(p.stdout.splitlines()):
        if line.startswith("{") and '"slab"' in line:
            d = json.loads(line)["slab"]
            d["wall_s"] = time.perf_counter() - t0
            return d
    return {"error": f"slab sub-run exited {p.returncode} without a result", "n_ranks": n}


# ---------------------------------------------------------------------------------------------------
# the CPU oracle (cpu_baseline leg, and the whole of --impl reference)
# ---------------------------------------------------------------------------------------------------
def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def run_oracle(workload: str, budget_s: float, steps: int | None, warmup: int = 0):
    """Times the oracle's multi-shift CG on the workload's inputs.  Returns (s_per_iter, cores, description, iters).
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


def run_oracle_extras():
    """SURVEY.md §8(d) "Oracle timing": the oracle's D_oe/D_eo pair at 32^4 -> ns/site on all cores and on one
    thread; the whole BASELINE config 2 solve (16^4) -> s/iter and iteration count."""
    import oracle
    out = {"nproc": os.cpu_count(), "cpu_model": cpu_model()}
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    cores = oracle.num_threads()
    L = gen.CONFIGS["config3_32^4"]["L"]
    U = gen.random_su3_links(L, device=dev).cpu().numpy()
    b = oracle.restrict(L, 0, gen.gaussian_field(L, device=dev).cpu().numpy())
    vh = b.shape[0]

    def pair_ns(reps):
        t = oracle.doe(L, U, b)
        oracle.deo(L, U, t)
        t0 = time.perf_counter()
        for _ in range(reps):
            t = oracle.doe(L, U, b)
            oracle.deo(L, U, t)
        return (time.perf_counter() - t0) / (2 * reps) / vh * 1e9

    out["dslash_ns_per_site"] = pair_ns(10)
    out["dslash_sample"] = f"10 x (D_oe, D_eo) at 32^4 on {cores} threads"
    try:
        oracle.set_num_threads(1)
        out["dslash_ns_per_site_1thread"] = pair_ns(2)
    finally:
        oracle.set_num_threads(cores)
    del U, b
    cfg = gen.CONFIGS["config2_16^4"]
    L = cfg["L"]
    U = gen.random_su3_links(L, device=dev).cpu().numpy()
    b = oracle.restrict(L, 0, gen.gaussian_field(L, device=dev).cpu().numpy())
    t0 = time.perf_counter()
    _, info = oracle.mshift_cg(L, U, cfg["mass"], b, cfg["shifts"], cfg["tol"])
    dt = time.perf_counter() - t0
    out["cg16_s_per_iter"] = dt / max(info["iters"], 1)
    out["cg16_iters"] = info["iters"]
    out["cg16_sample"] = f"whole config-2 solve (16^4, 8 shifts, tol 1e-10) on {cores} threads, {dt:.1f} s"
    return out


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
    ap.add_argument("--quick", action="store_true", help="skip the full solve, the 32^4 / small tables and the CPU baseline")
    ap.add_argument("--cpu-budget", type=float, default=20.0, help="seconds of oracle time for cpu_baseline")
    ap.add_argument("--with-slab", action="store_true",
                    help="also run the guarded slab sub-run when N = 1 (it always runs when N > 1)")
    ap.add_argument("--slab-check", action="store_true", help=argparse.SUPPRESS)
    ap.add_argument("--slab-comm", default="nccl", choices=["nccl", "p2p"],
                    help="transport of --parallel slab: the library's NCCL transport or its peer-memory transport")
    ap.add_argument("--plumbing-check", action="store_true", help=argparse.SUPPRESS)
    args = ap.parse_args()
    self_launch(args, sys.argv[1:])
    if args.plumbing_check:
        return run_plumbing_check(args)
    if args.slab_check:
        return run_slab_check(args)
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
              "step": "one multi-shift CG iteration (D_oe and D_eo with all sums and scalar products fused in, scalar "
                      "recurrences, 1/m of the block sweep over the x_i/p_i)",
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
    # the headline is complete on every rank; the other ranks are done (rank 0 alone finishes the report, and the slab
    # sub-run needs their GPUs idle)
    barrier(world)
    dist_teardown(world)
    if rank != 0:
        return 0
    K, W = args.steps, args.warmup
    peak, peak_src = res["peak"]
    ms_step = res["timed"]["ms_total"] / K
    value = ms_step * 1e-3 / world                     # replicas: N solves advance one iteration per ms_step
    ds_main = res["dslash"][lname][f"recon{args.recon}"]
    achieved = ds_main["gbs_dram_model"]
    ncu = NCU_DRAM_GB_PER_LAUNCH.get((args.workload, args.recon))
    read_ref = res.get("read_only_gbs")
    line = {
        "metric": "mshift_cg_s_per_iter", "value": value, "unit": "s/iter", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": config,
        "clocks": res["clocks"],
        "value_steady": res["steady"]["s_per_iter"] / world if "steady" in res else None,
        "e2e": {"value": res["e2e"]["ms_total"] * 1e-3 / K / world, "unit": "s/iter",
                "h2d_bytes_per_step": res["e2e"]["h2d"] / K, "d2h_bytes_per_step": res["e2e"]["d2h"] / K,
                "note": "lqcd_mshift_cg_host: pinned-host b in, 16 pinned-host solutions out, K iterations per call"},
        "gpu_launches": res["timed"]["launches_all"],
        "roofline": {"bound": "hbm", "kernel": f"dslash_kernel<{args.recon},0> (D_oe / D_eo) at {lname}",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": (ncu[0] + ncu[1]) * 1e9 if ncu else None,
                     "traffic_source": ncu[2] if ncu else None,
                     "peak_source": peak_src,
                     "bytes_per_launch": ds_main["dram_bytes_per_launch"], "us_per_launch": ds_main["us_per_application"],
                     "ns_per_site": ds_main["ns_per_site"],
                     "bytes_per_site": DSLASH_DRAM_MODEL[args.recon],
                     "achieved_algorithmic": ds_main["gbs_algorithmic"], "frac_algorithmic": ds_main["gbs_algorithmic"] / peak,
                     "algorithmic_bytes_per_site": DSLASH_BYTES[args.recon],
                     "frac_of_nominal_8000": achieved / 8000.0,
                     "read_only_reference_gbs": read_ref,
                     "frac_of_read_only_stream": achieved / read_ref if read_ref else None,
                     "note": "achieved = DRAM-compulsory bytes (8 links + 1 input vector + 1 output per site, SURVEY.md "
                             "8(d) 'each input once') / event time; peak is a COPY (half writes) while this kernel is 96 % "
                             "reads, hence frac slightly above 1 -- see frac_of_read_only_stream and frac_of_nominal_8000; "
                             "achieved_algorithmic also counts the 8 neighbour-vector reads that L1/L2 serve and is not an "
                             "HBM fraction"},
        "cg_roofline": {"bound": "hbm", "achieved": res["timed"]["gbs_dram"], "peak": peak, "unit": "GB/s",
                        "frac": res["timed"]["gbs_dram"] / peak,
                        "bytes_per_iteration": res["timed"]["bytes_dram"] / K, "n_active_mean": res["timed"]["n_active_mean"],
                        "shift_block": res["timed"]["shift_block"],
                        "steady_achieved": res["steady"]["gbs_dram"] if "steady" in res else None,
                        "method_equivalent_gbs": res["timed"]["gbs_method_equivalent"],
                        "note": "achieved = DRAM-compulsory bytes of the K timed iterations as the library runs them "
                                "(cg_dram_bytes: two fused operator sweeps + block sweeps, from the recorded freeze schedule) "
                                "/ time; method_equivalent_gbs = bytes of the method as the paper states it (SURVEY.md 8(d): "
                                "3600+192(n_act-1) B/site per iteration) / time, an equivalent rate, not an HBM fraction"},
        "dslash": res["dslash"],
    }
    if "e2e_rational" in res:
        er = res["e2e_rational"]
        line["e2e_rational"] = {"value": er["ms_total"] * 1e-3 / max(er["iters"], 1), "unit": "s/iter", "iters": er["iters"],
                                "h2d_bytes_per_step": er["h2d"] / max(er["iters"], 1),
                                "d2h_bytes_per_step": er["d2h"] / max(er["iters"], 1),
                                "device_s_per_iter": er["kernel_ms"] * 1e-3 / max(er["iters"], 1),
                                "note": "lqcd_rational_apply_host: pinned-host b in, ONE pinned-host vector out (the call "
                                        "the RHMC makes, PAPER.md:L82), K iterations per call, wall clock"}
    for key in ("full_solve", "dslash_slab", "cg_recon12", "cg_recon18", "next_rows", "small"):
        if key in res:
            line[key] = res[key]
    phase("GPU part done")
    if world > 1 or args.with_slab:
        # a sub-run takes ~30 s including start-up; the limits keep a hang from eating the time the driver allows the
        # whole bench (the headline line is printed after them)
        line["slab"] = guarded_slab_run(args, world, "nccl", timeout_s=300.0)
        line["slab_p2p"] = guarded_slab_run(args, world, "p2p", timeout_s=180.0)
        phase("slab sub-runs done")
    if not args.quick and world == 1:
        s_iter, cores, sample, _ = run_oracle(args.workload, budget_s=args.cpu_budget, steps=None)
        line["cpu_baseline"] = {"value": s_iter, "unit": "s/iter", "cores": cores, "kind": "oracle", "sample": sample}
        line["cpu_baseline"].update(run_oracle_extras())
    phase("CPU baseline done")
    print(json.dumps(line))
    return 0


if __name__ == "__main__":
    sys.exit(main())
