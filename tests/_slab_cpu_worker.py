"""Worker of tests/test_slab_host.py: the N>1 path on CPU.  W gloo ranks (2 or 4), the product's TorchTransport
(ring exchange of the faces, all-reduce) on CPU buffers, and the slab bookkeeping of the binding; the kernels are
replaced by the oracle applied to a whole-lattice vector that holds ONLY what the rank would have: its own slab
and the two faces it received.  If the exchange delivered the wrong face, or a face to the wrong side, the result
on the slab differs from the oracle's whole-lattice result."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np  # noqa: E402
import torch  # noqa: E402
import torch.distributed as dist  # noqa: E402

import oracle  # noqa: E402
from helpers import make_inputs, oracle_parity_vector, rel_l2  # noqa: E402
from paper_1801_01473_b200.binding import Lattice, TorchTransport  # noqa: E402

L = tuple(int(v) for v in sys.argv[1:5])
dist.init_process_group("gloo", init_method="env://")
rank, world = dist.get_rank(), dist.get_world_size()
tr = TorchTransport()
assert (tr.rank, tr.nranks) == (rank, world)

U, f = make_inputs(L)
b_soa, b_aos = oracle_parity_vector(L, f.numpy(), 0)
Vh = b_soa.shape[1]
face = L[0] * L[1] * L[2] // 2
a, b_ = Lattice.slab_range(L, rank, world)
k0, k1 = a // 2, b_ // 2

# what the library does in slab_dslash: pack the two faces of the local vector, exchange, use the halos
local = Lattice.slab_of_vector(torch.as_tensor(b_soa), L, rank, world)            # (3, Vh_loc, 2)
send_lo = local[:, :face].contiguous()
send_hi = local[:, -face:].contiguous()
recv_lo, recv_hi = torch.empty_like(send_lo), torch.empty_like(send_hi)
as_bytes = lambda t: t.view(-1).view(torch.uint8)
tr.exchange(as_bytes(send_lo), as_bytes(send_hi), as_bytes(recv_lo), as_bytes(recv_hi))

# whole-lattice vector holding only the slab and its two halos
have = np.zeros_like(b_soa)
have[:, k0:k1] = local.numpy()
lo0 = (k0 - face) % Vh
hi0 = k1 % Vh
if world > 1 or True:
    have[:, lo0:lo0 + face] = recv_lo.numpy()
    have[:, hi0:hi0 + face] = recv_hi.numpy()
out = oracle.aos_to_soa(oracle.doe(L, U.numpy(), oracle.soa_to_aos(have)))      # odd sites, whole lattice
ref = oracle.aos_to_soa(oracle.doe(L, U.numpy(), b_aos))
err = rel_l2(out[:, k0:k1], ref[:, k0:k1])
# the halos are exactly the neighbours' faces
halo_ok = bool(np.array_equal(recv_lo.numpy(), b_soa[:, lo0:lo0 + face]) and
               np.array_equal(recv_hi.numpy(), b_soa[:, hi0:hi0 + face]))

# scalar product: local partial, all-reduce, same bits everywhere
part = torch.tensor([float(np.sum(local.numpy() ** 2))], dtype=torch.float64)
tr.allreduce(part)
parts = [None] * world
dist.all_gather_object(parts, (float(part[0]), err, halo_ok))
if rank == 0:
    print("RESULT " + json.dumps(dict(
        err=max(p[1] for p in parts), halo_ok=all(p[2] for p in parts),
        sums_equal=all(p[0] == parts[0][0] for p in parts),
        sum_rel=abs(parts[0][0] - float(np.sum(b_soa ** 2))) / float(np.sum(b_soa ** 2)),
        exchanges=tr.n_exchange, allreduces=tr.n_allreduce)))
dist.barrier()
dist.destroy_process_group()
