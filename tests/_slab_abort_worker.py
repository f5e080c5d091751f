"""Worker of tests/test_gpu_slab.py::test_a_rank_that_stops_does_not_hang_the_others: 2 or 3 ranks under
torch.distributed.run (gloo for the set-up), all on cuda:0, the slab path over the peer-memory transport.  The LAST
rank sets up like the others and then does not take part in the solve:
    mode "abort": it calls lqcd_comm_abort (what a caller does before leaving early);
    mode "late" : it does nothing at all (a rank that hangs, or whose process is gone) -- it stays alive, asleep, so that
                  its window remains mapped: the others must give up by themselves after LQCD_OPT_COMM_TIMEOUT.
Every other rank must get LQCD_ECOMM from its solve, in bounded time, and again at once from the next call."""
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import torch  # noqa: E402
import torch.distributed as dist  # noqa: E402

import paper_1801_01473_b200 as lq  # noqa: E402
from helpers import make_inputs, oracle_parity_vector  # noqa: E402

MODE = sys.argv[1]
TIMEOUT_S = 3.0
L = (4, 4, 4, 12)
dist.init_process_group("gloo", init_method="env://")
rank, world = dist.get_rank(), dist.get_world_size()
torch.cuda.set_device(0)

U, f = make_inputs(L)
b_glob = torch.as_tensor(oracle_parity_vector(L, f.numpy(), 0)[0])
lat = lq.Lattice(L, mass=0.05, slab=(rank, world), comm="p2p")
lat.set_gauge(lq.Lattice.slab_of_links(U, L, rank, world).cuda())          # collective: everybody is connected after it
b = lq.Lattice.slab_of_vector(b_glob, L, rank, world).cuda()
shifts = [1e-3, 1e-1]
with torch.cuda.stream(torch.cuda.Stream()):
    x, info = lat.mshift_cg(b, shifts, 1e-10)                               # a healthy solve first
torch.cuda.synchronize()
assert info["status"] == 0
dist.barrier()

res = dict(rank=rank)
if rank == world - 1:
    if MODE == "abort":
        time.sleep(0.5)                  # the others are inside their solve by now, waiting for this rank
        lat.comm_abort()
else:
    lat.set_option(lq.LQCD_OPT_COMM_TIMEOUT, TIMEOUT_S if MODE == "late" else 60.0)
    t0 = time.time()
    codes = []
    with torch.cuda.stream(torch.cuda.Stream()):
        for _ in range(2):
            try:
                lat.mshift_cg(b, shifts, 1e-10)
                codes.append(0)
            except lq.LqcdError as e:
                codes.append(e.code)
                res.setdefault("text", str(e))
    res.update(codes=codes, seconds=time.time() - t0)
    torch.cuda.synchronize()             # this rank's streams have drained: nothing is left waiting
allres = [None] * world
dist.all_gather_object(allres, res)
if rank == 0:
    print("RESULT " + json.dumps(allres))
dist.barrier()                           # nobody unmaps a window another rank may still be writing to
lat.close()
dist.barrier()
dist.destroy_process_group()
