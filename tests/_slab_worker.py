"""Worker of tests/test_gpu_slab.py: 2 ranks under torch.distributed.run (gloo), both on cuda:0, the slab path with
the host-staged torch transport.  Rank 0 gathers the slabs and compares with the oracle on the whole lattice."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np  # noqa: E402
import torch  # noqa: E402
import torch.distributed as dist  # noqa: E402

import paper_1801_01473_b200 as lq  # noqa: E402
from helpers import make_inputs, oracle_parity_vector, rel_l2  # noqa: E402
import lqcd_inputs as gen  # noqa: E402
import oracle  # noqa: E402

L = tuple(int(v) for v in sys.argv[1:5])
RECON = int(sys.argv[6]) if len(sys.argv) > 6 else 18
# "torch": host-staged, ranks share cuda:0; "nccl": one GPU each; "p2p": peer-mapped windows, one GPU each when there
# are enough of them, else the ranks share the GPUs there are (CUDA IPC between processes on one device)
COMM = sys.argv[5] if len(sys.argv) > 5 else "torch"
dist.init_process_group("gloo", init_method="env://")
rank, world = dist.get_rank(), dist.get_world_size()
_lr = int(os.environ.get("LOCAL_RANK", "0"))
torch.cuda.set_device(_lr if COMM == "nccl" else (_lr % torch.cuda.device_count() if COMM == "p2p" else 0))

mass, tol, shifts = 0.05, 1e-10, [1e-3, 1e-2, 1e-1, 1.0]
U, f = make_inputs(L)                                   # every rank draws the same whole-lattice inputs
b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
b_glob = torch.as_tensor(b_soa)

lat = lq.Lattice(L, mass=mass, recon=RECON, slab=(rank, world), comm=COMM,
                 precisions=lq.LQCD_PREC_F64 | lq.LQCD_PREC_F32)
lat.set_gauge(lq.Lattice.slab_of_links(U, L, rank, world).cuda())
b = lq.Lattice.slab_of_vector(b_glob, L, rank, world).cuda()
with torch.cuda.stream(torch.cuda.Stream()):
    t = lat.doe(b)
    u = lat.deo(t)
    a = lat.mdagm(b, 0.3)
    x, info = lat.mshift_cg(b, shifts, tol)
    # the same operator with general U(1) phases (the angles of the t-links below the slab come from rank-1)
    theta = gen.random_u1_phases(L)
    a0, a1 = lq.Lattice.slab_range(L, rank, world)
    lat.set_u1_phases(theta[:, a0:a1].contiguous().cuda())
    tu = lat.doe(b)
    uu = lat.deo(tu)
    lat.set_u1_phases(None)
    # single precision on the same slabs
    t32 = lat.doe(b.float())
    x32, info32 = lat.mshift_cg(b.float(), shifts, 1e-5)
torch.cuda.synchronize()
assert lat.transport is None or lat.transport.error is None, lat.transport.error


def gather(v):
    """local parity vector (3, Vh_loc, 2) -> whole-lattice parity vector on rank 0"""
    v = v.cpu().contiguous()
    parts = [torch.empty_like(v) for _ in range(world)] if rank == 0 else None
    dist.gather(v, parts, dst=0)
    return torch.cat(parts, dim=1).numpy() if rank == 0 else None


tg, ug, ag = gather(t), gather(u), gather(a)
tug, uug = gather(tu), gather(uu)
t32g = gather(t32.double())
x32g = [gather(x32[i].double()) for i in range(len(shifts))]
xg = [gather(x[i]) for i in range(len(shifts))]
stats = [None] * world
dist.all_gather_object(stats, (info["iters"], info["freeze_iter"], info["rel_res"]))
if rank == 0:
    Un = U.numpy()
    t_ref = oracle.doe(L, Un, b_aos)
    u_ref = oracle.deo(L, Un, t_ref)
    a_ref = oracle.mdagm(L, Un, mass, 0.3, b_aos)
    x_ref, info_ref = oracle.mshift_cg(L, Un, mass, b_aos, shifts, tol)
    # DESIGN.md R9: beyond a few hundred iterations the count at which |r| crosses the threshold moves by a few under
    # one-ulp perturbations of the oracle itself; "+-1" is asked relative to the band the oracle spans
    counts = [info_ref["iters"]]
    if info_ref["iters"] > 300:
        counts.append(oracle.mshift_cg(L, Un, mass, b_aos, shifts, tol, sum_order=1)[1]["iters"])
        rng = np.random.default_rng(1234)
        for _ in range(2):
            bp = b_aos * (1.0 + rng.integers(-1, 2, size=b_aos.shape) * 2.0 ** -52)
            counts.append(oracle.mshift_cg(L, Un, mass, bp, shifts, tol)[1]["iters"])
    tu_ref = oracle.doe(L, Un, b_aos, theta=theta.numpy())
    uu_ref = oracle.deo(L, Un, tu_ref, theta=theta.numpy())
    res = dict(
        doe=rel_l2(oracle.soa_to_aos(tg), t_ref), deo=rel_l2(oracle.soa_to_aos(ug), u_ref),
        doe_f32=rel_l2(oracle.soa_to_aos(t32g), t_ref),
        x_f32=[rel_l2(oracle.soa_to_aos(x32g[i]), x_ref[i]) for i in range(len(shifts))],
        doe_u1=rel_l2(oracle.soa_to_aos(tug), tu_ref), deo_u1=rel_l2(oracle.soa_to_aos(uug), uu_ref),
        mdagm=rel_l2(oracle.soa_to_aos(ag), a_ref),
        x=[rel_l2(oracle.soa_to_aos(xg[i]), x_ref[i]) for i in range(len(shifts))],
        iters=info["iters"], iters_ref=info_ref["iters"], band=[min(counts), max(counts)],
        iters_equal_on_ranks=all(s[0] == stats[0][0] for s in stats),
        freeze_equal_on_ranks=all(s[1] == stats[0][1] and s[2] == stats[0][2] for s in stats),
        exchanges=lat.transport.n_exchange if lat.transport else None)
    print("RESULT " + json.dumps(res))
dist.barrier()          # nobody unmaps a window another rank may still be writing to
lat.close()
dist.barrier()
dist.destroy_process_group()
