"""lqcd_mdagm_static: the Eq. 2 operator for callers that cannot allocate device memory.

Some users of the library run inside a program that has already claimed the whole GPU for its own memory pool, so
a cudaMalloc made on their behalf fails; others sit on a path where the device-wide synchronisation that
cudaMalloc / cudaFree imply is not acceptable.  For them ``lqcd_mdagm_static`` does what ``lqcd_mdagm`` does, with
the odd-parity temporary in a 3 MiB buffer that is part of the library itself (include/lqcd.h).  That buffer is
shared by every call on the device and keeps what the previous call wrote, so what has to be shown is that

  * two calls in a row, with different inputs, shifts and even lattices, each give what ``lqcd_mdagm`` gives
    (same kernels, so the same bits are expected; the assertion uses the 1e-12 of the other operator tests);
  * the call really allocates nothing (free device memory is the same before and after);
  * a lattice beyond ``LQCD_STATIC_MAX_VH`` sites per parity is refused with a message that says so.

This file is named so that pytest collects it after every other one: with ``-x`` a failure here hides nothing.
The tests do not depend on what ran before them (the buffer's address is looked up once per process and device by
the library; a fresh process and a used one behave alike).
"""
import numpy as np
import pytest
import torch

from helpers import make_inputs, oracle_parity_vector, rel_l2

pytestmark = pytest.mark.gpu

TOL_D = 1e-12          # relative L2 of one operator application, as in test_gpu_parity.py


@pytest.fixture(scope="module")
def lq():
    import paper_1801_01473_b200 as lq
    lq.load_library()
    return lq


def cuda(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def _lattice(lq, L, recon, mass):
    U, f = make_inputs(L)
    lat = lq.Lattice(L, recon=recon)
    lat.set_gauge(U.cuda())
    lat.set_option(lq.LQCD_OPT_MASS, mass)
    b = cuda(oracle_parity_vector(L, f.numpy(), 0)[0])
    return lat, b


@pytest.mark.parametrize("recon", [18, 12])
def test_static_matches_mdagm_on_two_calls_in_a_row(lq, recon):
    # 16^4 is the largest hypercube the buffer holds (32768 of 65536 sites per parity); the second lattice is
    # smaller and ragged, so its call finds the leftovers of a larger one in the buffer
    lat_a, b_a = _lattice(lq, (16, 16, 16, 16), recon, 0.37)
    lat_b, b_b = _lattice(lq, (10, 6, 4, 14), recon, 0.05)
    b_a2 = torch.flip(b_a, dims=[1]).contiguous()            # a second, different input on the first lattice

    # the existing path first (this also has every kernel involved loaded before memory is measured)
    ref_1 = lat_a.mdagm(b_a, 0.11)
    ref_2 = lat_a.mdagm(b_a2, 2.5)
    ref_3 = lat_b.mdagm(b_b, 0.0)
    out_1, out_2, out_3 = torch.empty_like(b_a), torch.empty_like(b_a), torch.empty_like(b_b)
    torch.cuda.synchronize()

    lat_a.mdagm_static(b_a, out_1, 0.11)                     # first call on this device in a fresh process: set-up
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    lat_a.mdagm_static(b_a2, out_2, 2.5)                     # straight after it, other input and shift
    lat_b.mdagm_static(b_b, out_3, 0.0)                      # same stream, other context and lattice size
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]

    for out, ref in ((out_1, ref_1), (out_2, ref_2), (out_3, ref_3)):
        assert torch.isfinite(out).all()
        assert rel_l2(out.cpu().numpy(), ref.cpu().numpy()) <= TOL_D
        assert torch.equal(out, ref)                         # same launches on the same data: not one bit differs
    assert free_after == free_before, "lqcd_mdagm_static changed the amount of free device memory"
    # and the inputs are untouched
    assert torch.equal(b_a2, torch.flip(b_a, dims=[1]))
    lat_a.close()
    lat_b.close()


def test_static_refuses_what_does_not_fit(lq):
    L = (16, 16, 16, 34)                                     # 69632 sites per parity > 65536
    lat = lq.Lattice(L)
    assert lat.Vh > lq.LQCD_STATIC_MAX_VH
    v = torch.zeros((3, lat.Vh, 2), dtype=torch.float64, device="cuda")
    out = torch.full_like(v, 7.0)
    with pytest.raises(lq.LqcdError) as e:
        lat.mdagm_static(v, out, 0.0)
    assert e.value.code == lq.LQCD_EINVAL
    assert str(lat.Vh) in str(e.value) and str(lq.LQCD_STATIC_MAX_VH) in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                          # nothing was launched
    lat.close()

    # within the limit but without a gauge field: the usual error, still no launch
    lat = lq.Lattice((4, 4, 4, 4))
    v = torch.zeros((3, lat.Vh, 2), dtype=torch.float64, device="cuda")
    with pytest.raises(lq.LqcdError) as e:
        lat.mdagm_static(v, torch.empty_like(v), 0.0)
    assert e.value.code == lq.LQCD_ENOGAUGE
    lat.close()
