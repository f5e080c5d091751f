"""NEXT-3: the path on a 1-D slab decomposition along t (Alg. 1), against
the oracle applied to the WHOLE lattice.

One GPU is all there is here, so:
  * one rank, ring closed on itself, over the library's own NCCL transport (send/recv to self, all-reduce of one
    rank, CUDA graph with the NCCL operations captured) and over the host-staged torch transport: exercises the
    interior/border split, the halo buffers, the link halo and the unfused reductions;
  * two ranks as two processes that share the GPU, host-staged through gloo (tests/_slab_worker.py): exercises
    t_off != 0, the antiperiodic sign on the right rank, the ring order of the faces.  No kernel ever waits on
    another rank: the processes only block on the host;
  * the peer-memory transport (csrc/p2p.cuh): one rank (its own window as both neighbours), and two / four ranks as
    processes that share the GPU and map each other's windows over CUDA IPC.  Its waits are stream memory operations on
    the waiting rank's own memory, never a kernel.
"""
import json
import os
import signal
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch

import lqcd_inputs as gen
import oracle
import paper_1801_01473_b200 as lq
from helpers import make_inputs, oracle_parity_vector, rel_l2, soa_gpu_to_aos

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SHIFTS = [1e-3, 1e-2, 1e-1, 1.0]


@pytest.mark.parametrize("comm", ["nccl", "torch", "p2p"])
@pytest.mark.parametrize("L,recon", [((4, 6, 8, 10), 18), ((8, 4, 6, 2), 18), ((4, 4, 4, 4), 12)])
def test_one_rank_slab_operators_and_cg(L, recon, comm):
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    mass, tol = 0.05, 1e-10
    lat = lq.Lattice(L, mass=mass, recon=recon, slab=(0, 1), comm=comm)
    assert lq.lqcd_slab_info(lat.ctx) == (0, 0, 1, 0, L[3])
    lat.set_gauge(U.cuda())
    b = torch.as_tensor(b_soa).cuda()
    with torch.cuda.stream(torch.cuda.Stream()):
        t = lat.doe(b)
        u = lat.deo(t)
        a = lat.mdagm(b, 0.3)
        x, info = lat.mshift_cg(b, SHIFTS, tol)
    torch.cuda.synchronize()
    t_ref = oracle.doe(L, U.numpy(), b_aos)
    u_ref = oracle.deo(L, U.numpy(), t_ref)
    a_ref = oracle.mdagm(L, U.numpy(), mass, 0.3, b_aos)
    assert rel_l2(soa_gpu_to_aos(t), t_ref) <= 1e-12
    assert rel_l2(soa_gpu_to_aos(u), u_ref) <= 1e-12
    assert rel_l2(soa_gpu_to_aos(a), a_ref) <= 1e-12
    x_ref, info_ref = oracle.mshift_cg(L, U.numpy(), mass, b_aos, SHIFTS, tol)
    assert abs(info["iters"] - info_ref["iters"]) <= 1
    for i in range(len(SHIFTS)):
        assert rel_l2(soa_gpu_to_aos(x[i]), x_ref[i]) <= 1e-8
    if comm == "torch":
        assert lat.transport.error is None
        # two exchanges and two reductions per iteration (+ the link halo, 3 operator calls, |b|^2)
        assert lat.transport.n_exchange >= 2 * info["iters"] + 1 + 4
        assert lat.transport.n_allreduce >= 2 * info["iters"] + 1
    lat.close()


def test_one_rank_slab_equals_whole_lattice_bitwise():
    """Same arithmetic per site, whichever launch computes it: the operator on a one-rank slab is bit-identical to
    the whole-lattice kernel; so are the CG iterates up to the (different, still deterministic) summation order."""
    L = (8, 8, 8, 8)
    U, f = make_inputs(L)
    b_soa, _ = oracle_parity_vector(L, f.numpy(), 0)
    b = torch.as_tensor(b_soa).cuda()
    whole = lq.Lattice(L, mass=0.05)
    whole.set_gauge(U.cuda())
    slab = lq.Lattice(L, mass=0.05, slab=(0, 1), comm="nccl")
    slab.set_gauge(U.cuda())
    with torch.cuda.stream(torch.cuda.Stream()):
        t0, t1 = whole.doe(b), slab.doe(b)
        u0, u1 = whole.deo(t0), slab.deo(t1)
        x0, i0 = whole.mshift_cg(b, SHIFTS, 1e-10)
        x1, i1 = slab.mshift_cg(b, SHIFTS, 1e-10)
    torch.cuda.synchronize()
    assert torch.equal(t0, t1) and torch.equal(u0, u1)
    assert abs(i0["iters"] - i1["iters"]) <= 1
    for a, c in zip(x0, x1):
        assert rel_l2(a.cpu().numpy(), c.cpu().numpy()) <= 1e-9
    whole.close()
    slab.close()


def test_slab_f32_and_rational():
    L = (4, 4, 6, 8)
    U, f = make_inputs(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    lat = lq.Lattice(L, mass=0.1, slab=(0, 1), comm="nccl", precisions=lq.LQCD_PREC_F64 | lq.LQCD_PREC_F32)
    lat.set_gauge(U.cuda())
    b = torch.as_tensor(b_soa).cuda()
    alpha = [0.3, -0.2, 0.7, 0.1]
    with torch.cuda.stream(torch.cuda.Stream()):
        y = lat.rational_apply(b, 0.5, alpha, SHIFTS, 1e-10)[0]
        t32 = lat.doe(b.float())
    torch.cuda.synchronize()
    y_ref = oracle.rational_apply(L, U.numpy(), 0.1, b_aos, 0.5, alpha, SHIFTS, 1e-10)[0]
    assert rel_l2(soa_gpu_to_aos(y), y_ref) <= 1e-8
    Uf = U.float().double()
    t_ref = oracle.doe(L, Uf.numpy(), oracle.soa_to_aos(b.float().double().cpu().numpy()))
    assert rel_l2(soa_gpu_to_aos(t32.double()), t_ref) <= 2e-6
    lat.close()


def test_slab_with_u1_phases():
    L = (4, 6, 4, 6)
    U, f = make_inputs(L)
    theta = gen.random_u1_phases(L)
    b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
    lat = lq.Lattice(L, mass=0.1, slab=(0, 1), comm="nccl")
    lat.set_gauge(U.cuda())
    lat.set_u1_phases(theta.cuda())
    b = torch.as_tensor(b_soa).cuda()
    with torch.cuda.stream(torch.cuda.Stream()):
        t = lat.doe(b)
        u = lat.deo(t)
        x, info = lat.mshift_cg(b, SHIFTS, 1e-10)
    torch.cuda.synchronize()
    t_ref = oracle.doe(L, U.numpy(), b_aos, theta=theta.numpy())
    u_ref = oracle.deo(L, U.numpy(), t_ref, theta=theta.numpy())
    assert rel_l2(soa_gpu_to_aos(t), t_ref) <= 1e-12 and rel_l2(soa_gpu_to_aos(u), u_ref) <= 1e-12
    x_ref, info_ref = oracle.mshift_cg(L, U.numpy(), 0.1, b_aos, SHIFTS, 1e-10, theta=theta.numpy())
    assert abs(info["iters"] - info_ref["iters"]) <= 1
    assert max(rel_l2(soa_gpu_to_aos(x[i]), x_ref[i]) for i in range(len(SHIFTS))) <= 1e-8
    lat.close()


def test_slab_errors():
    assert not lq.lqcd_create_slab(4, 4, 4, 6, 0, 2)          # 3 time slices per rank: odd
    assert "even" in lq.lqcd_last_error(None)
    assert not lq.lqcd_create_slab(4, 4, 4, 8, 2, 2)
    ctx = lq.lqcd_create_slab(4, 4, 4, 8, 1, 2)
    assert ctx and lq.lqcd_slab_info(ctx) == (0, 1, 2, 4, 8)
    U = gen.random_su3_links((4, 4, 4, 4)).cuda()
    assert lq.lqcd_set_gauge(ctx, U.data_ptr()) == lq.LQCD_ECOMM      # no transport yet
    th = torch.zeros(4 * 256, dtype=torch.float64, device="cuda")
    assert lq.lqcd_set_u1_phases(ctx, th.data_ptr()) == lq.LQCD_ECOMM
    lq.lqcd_destroy(ctx)
    whole = lq.lqcd_create(4, 4, 4, 4)
    rc, nid = lq.lqcd_nccl_unique_id()
    assert rc == 0 and lq.lqcd_comm_init_nccl(whole, nid) == lq.LQCD_EINVAL
    lq.lqcd_destroy(whole)


def test_peer_memory_kernel_signal_fallback(monkeypatch):
    """The arrival words of a face set by a one-thread kernel instead of cuStreamWriteValue32 (what the transport falls
    back to when the driver refuses a stream memory operation on a peer-mapped address): same results, bit for bit."""
    L = (4, 4, 6, 8)
    U, f = make_inputs(L)
    b_soa, _ = oracle_parity_vector(L, f.numpy(), 0)
    b = torch.as_tensor(b_soa).cuda()
    out = []
    for flag in ("0", "1"):
        monkeypatch.setenv("LQCD_P2P_KERNEL_SIGNAL", flag)
        lat = lq.Lattice(L, mass=0.05, slab=(0, 1), comm="p2p")
        lat.set_gauge(U.cuda())
        with torch.cuda.stream(torch.cuda.Stream()):
            t = lat.doe(b)
            x, info = lat.mshift_cg(b, SHIFTS, 1e-10)
        torch.cuda.synchronize()
        out.append((t, x, info["iters"]))
        lat.close()
    assert torch.equal(out[0][0], out[1][0]) and out[0][2] == out[1][2]
    assert all(torch.equal(a, c) for a, c in zip(out[0][1], out[1][1]))


def test_peer_memory_transport_errors_and_determinism():
    """Argument checks of lqcd_p2p_export / lqcd_comm_init_p2p; and the solve over peer memory is bit-identical to the
    solve over NCCL on one rank (same launches, same order of every sum), launched plainly (no graph replays)."""
    whole = lq.lqcd_create(4, 4, 4, 4)
    rc, _ = lq.lqcd_p2p_export(whole)
    assert rc == lq.LQCD_EINVAL                                    # not a slab context
    lq.lqcd_destroy(whole)
    ctx = lq.lqcd_create_slab(4, 4, 4, 8, 0, 2)
    assert lq.lqcd_comm_init_p2p(ctx, bytes(2 * lq.LQCD_P2P_HANDLE_BYTES)) == lq.LQCD_ECOMM      # nothing exported yet
    rc, h = lq.lqcd_p2p_export(ctx)
    assert rc == 0 and len(h) == lq.LQCD_P2P_HANDLE_BYTES
    assert lq.lqcd_p2p_export(ctx)[0] == lq.LQCD_ECOMM             # one window per context
    assert lq.lqcd_comm_init_p2p(ctx, h + h) == lq.LQCD_ECOMM      # second entry is not rank 1's
    assert "rank order" in lq.lqcd_last_error(ctx)
    lq.lqcd_destroy(ctx)

    L = (4, 6, 4, 8)
    U, f = make_inputs(L)
    b_soa, _ = oracle_parity_vector(L, f.numpy(), 0)
    b = torch.as_tensor(b_soa).cuda()
    out = {}
    for comm in ("nccl", "p2p"):
        lat = lq.Lattice(L, mass=0.05, slab=(0, 1), comm=comm)
        lat.set_gauge(U.cuda())
        with torch.cuda.stream(torch.cuda.Stream()):
            t = lat.doe(b)
            x, info = lat.mshift_cg(b, SHIFTS, 1e-10)
        torch.cuda.synchronize()
        out[comm] = (t, x, info)
        lat.close()
    assert torch.equal(out["nccl"][0], out["p2p"][0])
    assert out["nccl"][2]["iters"] == out["p2p"][2]["iters"] and out["nccl"][2]["freeze_iter"] == out["p2p"][2]["freeze_iter"]
    for xa, xb in zip(out["nccl"][1], out["p2p"][1]):
        assert torch.equal(xa, xb)
    assert out["nccl"][2]["graph_replays"] > 0 and out["p2p"][2]["graph_replays"] == 0


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _run_ranks(world, L, comm, recon=18, timeout=600):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join("tests", "_slab_worker.py"), *[str(v) for v in L], comm, str(recon)]
    # its own process group, so that a rank that hangs can be killed together with its launcher
    proc = subprocess.Popen(cmd, cwd=ROOT, env=dict(os.environ, OMP_NUM_THREADS="4"), stdout=subprocess.PIPE,
                            stderr=subprocess.PIPE, text=True, start_new_session=True)
    try:
        stdout, stderr = proc.communicate(timeout=timeout)
    except subprocess.TimeoutExpired:
        os.killpg(proc.pid, signal.SIGKILL)
        stdout, stderr = proc.communicate()
        raise AssertionError(f"{world} ranks over {comm} timed out\n" + stdout[-2000:] + stderr[-3000:])
    out = subprocess.CompletedProcess(cmd, proc.returncode, stdout, stderr)
    assert out.returncode == 0, out.stdout[-2000:] + out.stderr[-3000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("RESULT ")]
    assert len(line) == 1, out.stdout[-2000:]
    r = json.loads(line[0][7:])
    assert r["doe"] <= 1e-12 and r["deo"] <= 1e-12 and r["mdagm"] <= 1e-12, r
    assert r["doe_u1"] <= 1e-12 and r["deo_u1"] <= 1e-12, r
    # single precision on the slabs (tolerances of tests/test_gpu_f32.py: 24 eps32 for the operator; the float solve
    # to 1e-5 against the double solutions)
    assert r["doe_f32"] <= 2e-6 and max(r["x_f32"]) <= 1e-3, r
    assert r["band"][0] - 1 <= r["iters"] <= r["band"][1] + 1 and r["iters_equal_on_ranks"], r
    assert max(r["x"]) <= 1e-8, r
    assert r["freeze_equal_on_ranks"], r


@pytest.mark.parametrize("L,recon", [((4, 6, 4, 8), 18), ((4, 4, 4, 4), 18), ((4, 4, 6, 8), 12)])
def test_two_ranks_share_the_gpu_host_staged(L, recon):
    _run_ranks(2, L, "torch", recon)


def test_four_ranks_share_the_gpu_host_staged():
    _run_ranks(4, (4, 4, 4, 8), "torch")            # two time slices per rank: no interior


@pytest.mark.parametrize("L,recon", [((4, 6, 4, 8), 18), ((4, 4, 6, 8), 12)])
def test_two_ranks_share_the_gpu_over_peer_memory(L, recon):
    """Two processes on one GPU map each other's windows over CUDA IPC: faces written into the neighbour's window,
    arrival flags by stream memory operations, scalar products through the windows' slots."""
    _run_ranks(2, L, "p2p", recon, timeout=300)


def test_four_ranks_share_the_gpu_over_peer_memory():
    _run_ranks(4, (4, 4, 4, 8), "p2p", timeout=300)     # two time slices per rank: no interior, four-way all-reduce


@pytest.mark.parametrize("mode,world", [("abort", 2), ("abort", 3), ("late", 2)])
def test_a_rank_that_stops_does_not_hang_the_others(mode, world):
    """Peer-memory transport: the ranks wait for each other with stream operations on flag words, so a rank that stops
    calling would leave the others waiting for ever.  The last rank sets up, takes part in one solve, then either calls
    lqcd_comm_abort or just stays away (tests/_slab_abort_worker.py).  Every other rank -- with three ranks also the
    one that is not the quitter's... every rank is a neighbour on a ring of three, but rank 0 and 1 also wait for each
    other -- must return LQCD_ECOMM from its solve in bounded time (at once after an abort, after
    LQCD_OPT_COMM_TIMEOUT = 3 s for a silent peer), must get LQCD_ECOMM again at once from the next call, and its
    streams must drain."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join("tests", "_slab_abort_worker.py"), mode]
    proc = subprocess.Popen(cmd, cwd=ROOT, env=dict(os.environ, OMP_NUM_THREADS="4"), stdout=subprocess.PIPE,
                            stderr=subprocess.PIPE, text=True, start_new_session=True)
    try:
        stdout, stderr = proc.communicate(timeout=240)
    except subprocess.TimeoutExpired:
        os.killpg(proc.pid, signal.SIGKILL)
        stdout, stderr = proc.communicate()
        raise AssertionError(f"{mode}: the ranks hung\n" + stdout[-2000:] + stderr[-3000:])
    assert proc.returncode == 0, stdout[-2000:] + stderr[-3000:]
    line = [l for l in stdout.splitlines() if l.startswith("RESULT ")]
    assert len(line) == 1, stdout[-2000:]
    res = json.loads(line[0][7:])
    assert len(res) == world
    for r in res[:-1]:
        assert r["codes"] == [-8, -8], res                        # LQCD_ECOMM, twice
        assert r["seconds"] < (30.0 if mode == "late" else 20.0), res
        if mode == "late":
            assert r["seconds"] >= 2.5 and "LQCD_OPT_COMM_TIMEOUT" in r["text"], res


@pytest.mark.parametrize("comm", ["nccl", "p2p"])
@pytest.mark.parametrize("world,L", [(2, (8, 8, 8, 8)), (4, (4, 6, 8, 16))])
def test_ranks_on_their_own_gpus_over_nccl(world, L, comm):
    """The production transports between GPUs: needs `world` devices, skipped on a one-GPU box."""
    if torch.cuda.device_count() < world:
        pytest.skip(f"needs {world} GPUs")
    _run_ranks(world, L, comm)
