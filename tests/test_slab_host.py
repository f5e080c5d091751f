"""Host side of the slab path (NEXT-3) without a GPU: the ring exchange and the all-reduce of the product's
TorchTransport over gloo with 2 and 4 ranks, the slab bookkeeping, and argument checks of lqcd_create_slab."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world,L", [(2, (4, 4, 6, 8)), (2, (4, 4, 4, 4)), (4, (4, 6, 4, 8))])
def test_ring_exchange_and_allreduce_over_gloo(world, L):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join("tests", "_slab_cpu_worker.py"), *[str(v) for v in L]]
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="2")
    out = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stdout[-1500:] + out.stderr[-3000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("RESULT ")]
    assert len(line) == 1
    r = json.loads(line[0][7:])
    assert r["halo_ok"] and r["err"] <= 1e-14, r
    assert r["sums_equal"] and r["sum_rel"] <= 1e-14, r
    assert r["exchanges"] == 1 and r["allreduces"] == 1


def test_single_process_ring_closes_on_itself():
    from paper_1801_01473_b200.binding import TorchTransport
    tr = TorchTransport()
    assert (tr.rank, tr.nranks) == (0, 1)
    lo, hi = torch.arange(8, dtype=torch.uint8), torch.arange(8, 16, dtype=torch.uint8)
    rlo, rhi = torch.zeros(8, dtype=torch.uint8), torch.zeros(8, dtype=torch.uint8)
    tr.exchange(lo, hi, rlo, rhi)
    assert torch.equal(rlo, hi) and torch.equal(rhi, lo)      # below me is my own top slice, above me my bottom one
    # through the C callback signature
    import ctypes
    a = (ctypes.c_uint8 * 4)(1, 2, 3, 4)
    b = (ctypes.c_uint8 * 4)(5, 6, 7, 8)
    c, d = (ctypes.c_uint8 * 4)(), (ctypes.c_uint8 * 4)()
    rc = tr.ops.exchange(None, ctypes.addressof(a), ctypes.addressof(b), ctypes.addressof(c), ctypes.addressof(d), 4, None)
    assert rc == 0 and list(c) == [5, 6, 7, 8] and list(d) == [1, 2, 3, 4]
    v = (ctypes.c_double * 2)(1.5, 2.5)
    assert tr.ops.allreduce_sum(None, v, 2, None) == 0 and list(v) == [1.5, 2.5]


def test_slab_bookkeeping():
    from paper_1801_01473_b200.binding import Lattice
    L = (4, 6, 2, 8)
    V = 4 * 6 * 2 * 8
    ranges = [Lattice.slab_range(L, r, 4) for r in range(4)]
    assert ranges[0][0] == 0 and ranges[-1][1] == V
    assert all(ranges[i][1] == ranges[i + 1][0] for i in range(3))
    links = torch.arange(4 * V, dtype=torch.float64).reshape(4, V, 1, 1, 1).expand(4, V, 3, 3, 2)
    s = Lattice.slab_of_links(links, L, 2, 4)
    assert s.shape == (4, V // 4, 3, 3, 2) and s.is_contiguous()
    assert float(s[1, 0, 0, 0, 0]) == V + 2 * (V // 4)
    v = torch.arange(3 * (V // 2), dtype=torch.float64).reshape(3, V // 2, 1).expand(3, V // 2, 2)
    sv = Lattice.slab_of_vector(v, L, 3, 4)
    assert sv.shape == (3, V // 8, 2) and float(sv[2, 0, 0]) == 2 * (V // 2) + 3 * (V // 8)


def test_create_slab_argument_checks():
    import paper_1801_01473_b200 as lq
    assert not lq.lqcd_create_slab(4, 4, 4, 6, 0, 2)
    assert "even number of time slices" in lq.lqcd_last_error(None)
    assert not lq.lqcd_create_slab(4, 4, 4, 8, 2, 2)
    assert "not a valid slab" in lq.lqcd_last_error(None)
    assert not lq.lqcd_create_slab(4, 4, 4, 8, 0, 3)
    rc, nid = lq.lqcd_nccl_unique_id()
    assert rc in (lq.LQCD_OK, lq.LQCD_ECOMM) and len(nid) == lq.LQCD_NCCL_ID_BYTES
