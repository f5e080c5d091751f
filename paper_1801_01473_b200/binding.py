"""ctypes binding of include/lqcd.h -- same names, argument marshalling only."""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

HERE = os.path.dirname(os.path.abspath(__file__))

# ---- constants of include/lqcd.h ---------------------------------------------------------------------
LQCD_OK, LQCD_EINVAL, LQCD_ENOGAUGE, LQCD_ENOMEM, LQCD_ECUDA = 0, -1, -2, -3, -4
LQCD_ENOCONV, LQCD_EBREAKDOWN, LQCD_ENOTSU3, LQCD_ECOMM = -5, -6, -7, -8
LQCD_NCCL_ID_BYTES = 128
LQCD_P2P_HANDLE_BYTES = 96
LQCD_STATIC_MAX_VH = 65536       # lqcd_mdagm_static: sites per parity its built-in buffer holds
LQCD_OPT_MASS, LQCD_OPT_ANTIPERIODIC_T, LQCD_OPT_RECON, LQCD_OPT_MAX_ITER = 0, 1, 2, 3
LQCD_OPT_CHECK_EVERY, LQCD_OPT_USE_GRAPH, LQCD_OPT_LINK_PRECISIONS, LQCD_OPT_SHIFT_BLOCK = 4, 5, 6, 7
LQCD_OPT_PERSISTENT = 8
LQCD_PREC_F64, LQCD_PREC_F32 = 1, 2
LQCD_STAT_ITERS, LQCD_STAT_REL_RES, LQCD_STAT_FREEZE_ITER, LQCD_STAT_BASE_SHIFT = 0, 1, 2, 3
LQCD_STAT_GPU_LAUNCHES, LQCD_STAT_SOLVE_MS, LQCD_STAT_RELIABLE_UPDATES, LQCD_STAT_GRAPH_REPLAYS = 4, 5, 6, 7
LQCD_OPT_COMM_TIMEOUT = 9          # seconds a solve over the peer-memory transport waits for its peers (0: for ever)
LQCD_STAT_SOLVER_PATH = 8          # 0 = plain launches, 1 = CUDA-graph replays, 2 = persistent kernel

_ERRNAMES = {0: "LQCD_OK", -1: "LQCD_EINVAL", -2: "LQCD_ENOGAUGE", -3: "LQCD_ENOMEM", -4: "LQCD_ECUDA",
             -5: "LQCD_ENOCONV", -6: "LQCD_EBREAKDOWN", -7: "LQCD_ENOTSU3", -8: "LQCD_ECOMM"}

_vp, _dp, _sz, _i, _d = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int, ctypes.c_double
_pd = ctypes.POINTER(ctypes.c_double)
_pi = ctypes.POINTER(ctypes.c_int)

# lqcd_comm_ops of include/lqcd.h
EXCHANGE_FN = ctypes.CFUNCTYPE(_i, _vp, _vp, _vp, _vp, _vp, _sz, _vp)
ALLREDUCE_FN = ctypes.CFUNCTYPE(_i, _vp, _pd, _i, _vp)


class lqcd_comm_ops(ctypes.Structure):
    _fields_ = [("user", _vp), ("exchange", EXCHANGE_FN), ("allreduce_sum", ALLREDUCE_FN),
                ("host_staged", _i), ("graph_safe", _i)]


# every symbol include/lqcd.h declares: name -> (restype, argtypes)
EXPORTS = {
    "lqcd_create": (_vp, [_i, _i, _i, _i]),
    "lqcd_destroy": (None, [_vp]),
    "lqcd_set_stream": (_i, [_vp, _vp]),
    "lqcd_set_option": (_i, [_vp, _i, _d]),
    "lqcd_get_option": (_i, [_vp, _i, _pd]),
    "lqcd_workspace_bytes": (_sz, [_vp, _i]),
    "lqcd_set_workspace": (_i, [_vp, _vp, _sz]),
    "lqcd_set_gauge": (_i, [_vp, _dp]),
    "lqcd_set_gauge_host": (_i, [_vp, _dp]),
    "lqcd_set_u1_phases": (_i, [_vp, _dp]),
    "lqcd_set_u1_phases_host": (_i, [_vp, _dp]),
    "lqcd_doe": (_i, [_vp, _dp, _dp]),
    "lqcd_deo": (_i, [_vp, _dp, _dp]),
    "lqcd_doe_host": (_i, [_vp, _dp, _dp]),
    "lqcd_deo_host": (_i, [_vp, _dp, _dp]),
    "lqcd_mdagm": (_i, [_vp, _dp, _dp, _d]),
    "lqcd_mdagm_static": (_i, [_vp, _dp, _dp, _d]),
    "lqcd_mshift_cg": (_i, [_vp, _dp, _pd, _i, _d, ctypes.POINTER(ctypes.c_void_p)]),
    "lqcd_mshift_cg_host": (_i, [_vp, _dp, _pd, _i, _d, ctypes.POINTER(ctypes.c_void_p)]),
    "lqcd_mshift_cg_mixed": (_i, [_vp, _dp, _pd, _i, _d, ctypes.POINTER(ctypes.c_void_p)]),
    "lqcd_rational_apply": (_i, [_vp, _dp, _d, _pd, _pd, _i, _d, _dp]),
    "lqcd_rational_apply_host": (_i, [_vp, _dp, _d, _pd, _pd, _i, _d, _dp]),
    "lqcd_doe_f32": (_i, [_vp, _dp, _dp]),
    "lqcd_deo_f32": (_i, [_vp, _dp, _dp]),
    "lqcd_doe_f32_host": (_i, [_vp, _dp, _dp]),
    "lqcd_deo_f32_host": (_i, [_vp, _dp, _dp]),
    "lqcd_mdagm_f32": (_i, [_vp, _dp, _dp, _d]),
    "lqcd_mshift_cg_f32": (_i, [_vp, _dp, _pd, _i, _d, ctypes.POINTER(ctypes.c_void_p)]),
    "lqcd_mshift_cg_f32_host": (_i, [_vp, _dp, _pd, _i, _d, ctypes.POINTER(ctypes.c_void_p)]),
    "lqcd_rational_apply_f32": (_i, [_vp, _dp, _d, _pd, _pd, _i, _d, _dp]),
    "lqcd_get_stat": (_i, [_vp, _i, _i, _pd]),
    "lqcd_pack_vector": (_i, [_vp, _i, _dp, _dp]),
    "lqcd_unpack_vector": (_i, [_vp, _i, _dp, _dp]),
    "lqcd_pack_vector_f32": (_i, [_vp, _i, _dp, _dp]),
    "lqcd_unpack_vector_f32": (_i, [_vp, _i, _dp, _dp]),
    "lqcd_last_error": (ctypes.c_char_p, [_vp]),
    "lqcd_create_slab": (_vp, [_i, _i, _i, _i, _i, _i]),
    "lqcd_set_comm": (_i, [_vp, ctypes.POINTER(lqcd_comm_ops)]),
    "lqcd_nccl_unique_id": (_i, [_vp]),
    "lqcd_comm_init_nccl": (_i, [_vp, _vp]),
    "lqcd_p2p_export": (_i, [_vp, _vp]),
    "lqcd_comm_init_p2p": (_i, [_vp, _vp]),
    "lqcd_slab_info": (_i, [_vp, _pi, _pi, _pi, _pi]),
    "lqcd_comm_abort": (_i, [_vp]),
}

_lib = None


def library_path() -> str:
    return os.path.join(HERE, "liblqcd_b200.so")


def load_library():
    """dlopen liblqcd_b200.so (building it with nvcc if it is missing or was built from other sources than the
    ones in the tree now).  Raises if that fails: there is no other implementation to fall back to."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    from .build import build
    build()                              # returns at once when the library matches the sources
    lib = ctypes.CDLL(path)
    for name, (res, args) in EXPORTS.items():
        fn = getattr(lib, name)          # AttributeError if the symbol is missing
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


class LqcdError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"{_ERRNAMES.get(code, code)}: {text}")
        self.code = code


# ---- the C functions under their own names (raw pointers as ints) ------------------------------------
def lqcd_create(Lx, Ly, Lz, Lt):
    return load_library().lqcd_create(int(Lx), int(Ly), int(Lz), int(Lt))


def lqcd_destroy(ctx):
    load_library().lqcd_destroy(ctx)


def lqcd_set_stream(ctx, cuda_stream):
    return load_library().lqcd_set_stream(ctx, cuda_stream)


def lqcd_set_option(ctx, key, value):
    return load_library().lqcd_set_option(ctx, int(key), float(value))


def lqcd_get_option(ctx, key):
    out = ctypes.c_double()
    rc = load_library().lqcd_get_option(ctx, int(key), ctypes.byref(out))
    return rc, out.value


def lqcd_workspace_bytes(ctx, nshift):
    return load_library().lqcd_workspace_bytes(ctx, int(nshift))


def lqcd_set_workspace(ctx, dev, nbytes):
    return load_library().lqcd_set_workspace(ctx, dev, int(nbytes))


def lqcd_set_gauge(ctx, links):
    return load_library().lqcd_set_gauge(ctx, links)


def lqcd_set_gauge_host(ctx, links):
    return load_library().lqcd_set_gauge_host(ctx, links)


def lqcd_set_u1_phases(ctx, theta):
    return load_library().lqcd_set_u1_phases(ctx, theta)


def lqcd_set_u1_phases_host(ctx, theta):
    return load_library().lqcd_set_u1_phases_host(ctx, theta)


def lqcd_doe(ctx, out_odd, in_even):
    return load_library().lqcd_doe(ctx, out_odd, in_even)


def lqcd_deo(ctx, out_even, in_odd):
    return load_library().lqcd_deo(ctx, out_even, in_odd)


def lqcd_doe_host(ctx, out_odd, in_even):
    return load_library().lqcd_doe_host(ctx, out_odd, in_even)


def lqcd_deo_host(ctx, out_even, in_odd):
    return load_library().lqcd_deo_host(ctx, out_even, in_odd)


def lqcd_mdagm(ctx, out_even, in_even, sigma):
    return load_library().lqcd_mdagm(ctx, out_even, in_even, float(sigma))


def lqcd_doe_f32(ctx, out_odd, in_even):
    return load_library().lqcd_doe_f32(ctx, out_odd, in_even)


def lqcd_deo_f32(ctx, out_even, in_odd):
    return load_library().lqcd_deo_f32(ctx, out_even, in_odd)


def lqcd_doe_f32_host(ctx, out_odd, in_even):
    return load_library().lqcd_doe_f32_host(ctx, out_odd, in_even)


def lqcd_deo_f32_host(ctx, out_even, in_odd):
    return load_library().lqcd_deo_f32_host(ctx, out_even, in_odd)


def lqcd_comm_abort(ctx):
    return load_library().lqcd_comm_abort(ctx)


def lqcd_mdagm_static(ctx, out_even, in_even, sigma):
    return load_library().lqcd_mdagm_static(ctx, out_even, in_even, float(sigma))


def lqcd_mdagm_f32(ctx, out_even, in_even, sigma):
    return load_library().lqcd_mdagm_f32(ctx, out_even, in_even, float(sigma))


def _cg_args(shifts, x_ptrs):
    n = len(shifts)
    sh = (ctypes.c_double * n)(*[float(s) for s in shifts])
    xs = (ctypes.c_void_p * n)(*[int(p) for p in x_ptrs])
    return n, sh, xs


def lqcd_mshift_cg(ctx, b_even, shifts: Sequence[float], tol: float, x_ptrs: Sequence[int]):
    n, sh, xs = _cg_args(shifts, x_ptrs)
    return load_library().lqcd_mshift_cg(ctx, b_even, sh, n, float(tol), xs)


def lqcd_mshift_cg_host(ctx, b_even, shifts: Sequence[float], tol: float, x_ptrs: Sequence[int]):
    n, sh, xs = _cg_args(shifts, x_ptrs)
    return load_library().lqcd_mshift_cg_host(ctx, b_even, sh, n, float(tol), xs)


def lqcd_mshift_cg_mixed(ctx, b_even, shifts: Sequence[float], tol: float, x_ptrs: Sequence[int]):
    n, sh, xs = _cg_args(shifts, x_ptrs)
    return load_library().lqcd_mshift_cg_mixed(ctx, b_even, sh, n, float(tol), xs)


def lqcd_mshift_cg_f32(ctx, b_even, shifts: Sequence[float], tol: float, x_ptrs: Sequence[int]):
    n, sh, xs = _cg_args(shifts, x_ptrs)
    return load_library().lqcd_mshift_cg_f32(ctx, b_even, sh, n, float(tol), xs)


def lqcd_mshift_cg_f32_host(ctx, b_even, shifts: Sequence[float], tol: float, x_ptrs: Sequence[int]):
    n, sh, xs = _cg_args(shifts, x_ptrs)
    return load_library().lqcd_mshift_cg_f32_host(ctx, b_even, sh, n, float(tol), xs)


def _rational(name, ctx, b_even, alpha0, alpha, shifts, tol, y_even):
    n = len(shifts)
    assert len(alpha) == n
    al = (ctypes.c_double * n)(*[float(a) for a in alpha])
    sh = (ctypes.c_double * n)(*[float(s) for s in shifts])
    return getattr(load_library(), name)(ctx, b_even, float(alpha0), al, sh, n, float(tol), y_even)


def lqcd_rational_apply(ctx, b_even, alpha0: float, alpha: Sequence[float], shifts: Sequence[float], tol: float,
                        y_even, host: bool = False):
    return _rational("lqcd_rational_apply_host" if host else "lqcd_rational_apply", ctx, b_even, alpha0, alpha,
                     shifts, tol, y_even)


def lqcd_rational_apply_f32(ctx, b_even, alpha0, alpha, shifts, tol, y_even):
    return _rational("lqcd_rational_apply_f32", ctx, b_even, alpha0, alpha, shifts, tol, y_even)


def lqcd_rational_apply_host(ctx, b_even, alpha0, alpha, shifts, tol, y_even):
    return lqcd_rational_apply(ctx, b_even, alpha0, alpha, shifts, tol, y_even, host=True)


def lqcd_get_stat(ctx, key, idx=0):
    out = ctypes.c_double()
    rc = load_library().lqcd_get_stat(ctx, int(key), int(idx), ctypes.byref(out))
    return rc, out.value


def lqcd_pack_vector(ctx, parity, site_field, parity_vector):
    return load_library().lqcd_pack_vector(ctx, int(parity), site_field, parity_vector)


def lqcd_unpack_vector(ctx, parity, parity_vector, site_field):
    return load_library().lqcd_unpack_vector(ctx, int(parity), parity_vector, site_field)


def lqcd_pack_vector_f32(ctx, parity, site_field, parity_vector):
    return load_library().lqcd_pack_vector_f32(ctx, int(parity), site_field, parity_vector)


def lqcd_unpack_vector_f32(ctx, parity, parity_vector, site_field):
    return load_library().lqcd_unpack_vector_f32(ctx, int(parity), parity_vector, site_field)


def lqcd_last_error(ctx) -> str:
    s = load_library().lqcd_last_error(ctx)
    return s.decode() if s else ""


def lqcd_create_slab(Lx, Ly, Lz, Lt_global, rank, nranks):
    return load_library().lqcd_create_slab(int(Lx), int(Ly), int(Lz), int(Lt_global), int(rank), int(nranks))


def lqcd_set_comm(ctx, ops: "lqcd_comm_ops"):
    return load_library().lqcd_set_comm(ctx, ctypes.byref(ops))


def lqcd_nccl_unique_id():
    """-> (rc, 128 bytes)"""
    buf = ctypes.create_string_buffer(LQCD_NCCL_ID_BYTES)
    rc = load_library().lqcd_nccl_unique_id(ctypes.cast(buf, _vp))
    return rc, buf.raw


def lqcd_comm_init_nccl(ctx, nccl_id: bytes):
    assert len(nccl_id) == LQCD_NCCL_ID_BYTES
    buf = ctypes.create_string_buffer(bytes(nccl_id), LQCD_NCCL_ID_BYTES)
    return load_library().lqcd_comm_init_nccl(ctx, ctypes.cast(buf, _vp))


def lqcd_p2p_export(ctx):
    """-> (rc, LQCD_P2P_HANDLE_BYTES bytes)"""
    buf = ctypes.create_string_buffer(LQCD_P2P_HANDLE_BYTES)
    rc = load_library().lqcd_p2p_export(ctx, ctypes.cast(buf, _vp))
    return rc, buf.raw


def lqcd_comm_init_p2p(ctx, handles: bytes):
    """``handles``: the LQCD_P2P_HANDLE_BYTES of every rank, concatenated in rank order"""
    assert len(handles) % LQCD_P2P_HANDLE_BYTES == 0
    buf = ctypes.create_string_buffer(bytes(handles), len(handles))
    return load_library().lqcd_comm_init_p2p(ctx, ctypes.cast(buf, _vp))


def lqcd_slab_info(ctx):
    """-> (rc, rank, nranks, t_offset, Lt_global)"""
    v = [ctypes.c_int(0) for _ in range(4)]
    rc = load_library().lqcd_slab_info(ctx, *[ctypes.byref(x) for x in v])
    return (rc,) + tuple(x.value for x in v)


# ---- a transport on top of torch.distributed (include/lqcd.h: lqcd_comm_ops, host_staged = 1) ----------------
class TorchTransport:
    """The two communication steps of the slab path (ring exchange of the faces along t, all-reduce of a scalar
    product) carried by ``torch.distributed`` on HOST buffers -- any backend that moves CPU tensors (gloo).  The
    library stages device data through pinned host memory around the calls, so ranks never wait on one another
    inside a kernel and may even share a GPU (tests).  The production transport is ``lqcd_comm_init_nccl``.

    Messages that travel up the ring (to rank+1) carry tag 1, those that travel down tag 2: with two ranks both
    neighbours are the same peer and only the tag tells the two faces apart."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist = dist
        self.group = group
        if dist.is_initialized():
            self.rank, self.nranks = dist.get_rank(group), dist.get_world_size(group)
        else:                       # a single process: the ring closes on itself
            self.rank, self.nranks = 0, 1
        self.error = None
        self._fx = EXCHANGE_FN(self._exchange)
        self._fa = ALLREDUCE_FN(self._allreduce)
        self.ops = lqcd_comm_ops(None, self._fx, self._fa, 1, 0)
        self.n_exchange = 0
        self.n_allreduce = 0

    @staticmethod
    def _bytes(ptr, n):
        import numpy as np
        import torch
        return torch.from_numpy(np.ctypeslib.as_array((ctypes.c_uint8 * n).from_address(ptr)))

    def exchange(self, send_lo, send_hi, recv_lo, recv_hi):
        """uint8 CPU tensors of equal size: send_lo -> rank-1, send_hi -> rank+1; recv_lo <- rank-1's send_hi,
        recv_hi <- rank+1's send_lo."""
        dist, g = self.dist, self.group
        up, dn = (self.rank + 1) % self.nranks, (self.rank - 1) % self.nranks
        self.n_exchange += 1
        if self.nranks == 1:
            recv_lo.copy_(send_hi)
            recv_hi.copy_(send_lo)
            return
        reqs = [dist.irecv(recv_lo, src=dn, group=g, tag=1), dist.irecv(recv_hi, src=up, group=g, tag=2),
                dist.isend(send_hi, dst=up, group=g, tag=1), dist.isend(send_lo, dst=dn, group=g, tag=2)]
        for r in reqs:
            r.wait()

    def allreduce(self, buf):
        self.n_allreduce += 1
        if self.nranks > 1:
            self.dist.all_reduce(buf, op=self.dist.ReduceOp.SUM, group=self.group)

    def _exchange(self, user, slo, shi, rlo, rhi, nbytes, stream):
        try:
            self.exchange(self._bytes(slo, nbytes), self._bytes(shi, nbytes), self._bytes(rlo, nbytes),
                          self._bytes(rhi, nbytes))
            return 0
        except Exception as e:  # an exception must not cross the C frame
            self.error = e
            return 1

    def _allreduce(self, user, buf, n, stream):
        try:
            import numpy as np
            import torch
            self.allreduce(torch.from_numpy(np.ctypeslib.as_array(buf, shape=(n,))))
            return 0
        except Exception as e:
            self.error = e
            return 1


# ---- torch-tensor convenience wrapper ------------------------------------------------------------------
class Lattice:
    """One lqcd_ctx.  float64 tensors go to the double entry points, float32 tensors to the ``*_f32`` ones
    (``precisions`` says which copies of the links ``set_gauge`` stores); device tensors go to the device
    entry points on torch's current stream, CPU tensors to the ``*_host`` entry points (the copies happen
    inside the call)."""

    # options applied to every context at creation, {key: value} (tests use it to run whole modules on one solver path)
    default_options: dict = {}

    def __init__(self, L: Sequence[int], mass: float = 0.0, antiperiodic: bool = True, recon: int = 18,
                 precisions: int = LQCD_PREC_F64, slab: Optional[Sequence[int]] = None, comm: Optional[str] = None,
                 group=None):
        """``slab=(rank, nranks)``: this process owns time slices [rank*Lt/nranks, (rank+1)*Lt/nranks) of the
        lattice ``L`` (include/lqcd.h, slab decomposition); all tensors are then those of the local lattice
        ``self.L`` = (Lx, Ly, Lz, Lt/nranks).  ``comm``: "nccl" (the library's own NCCL communicator; the id is
        handed round with ``torch.distributed``), "p2p" (the library's peer-memory transport; the window handles are
        handed round with ``torch.distributed``) or "torch" (:class:`TorchTransport`, host-staged)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1801_01473_b200 needs a CUDA device (there is no CPU fallback)")
        self._torch = torch
        self.L_global = tuple(int(v) for v in L)
        self.transport = None
        if slab is None:
            self.L = self.L_global
            self.ctx = lqcd_create(*self.L)
        else:
            rank, nranks = int(slab[0]), int(slab[1])
            self.ctx = lqcd_create_slab(*self.L_global, rank, nranks)
            self.L = self.L_global[:3] + (self.L_global[3] // max(nranks, 1),)
        if not self.ctx:
            raise LqcdError(LQCD_EINVAL, lqcd_last_error(None))
        self.V = self.L[0] * self.L[1] * self.L[2] * self.L[3]
        self.Vh = self.V // 2
        if slab is not None:
            self._init_comm(comm or "nccl", rank, nranks, group)
        for key, value in self.default_options.items():
            self.set_option(key, value)
        self.set_option(LQCD_OPT_MASS, mass)
        self.set_option(LQCD_OPT_ANTIPERIODIC_T, 1.0 if antiperiodic else 0.0)
        self.set_option(LQCD_OPT_RECON, recon)
        self.set_option(LQCD_OPT_LINK_PRECISIONS, precisions)

    def _init_comm(self, comm: str, rank: int, nranks: int, group):
        torch = self._torch
        if comm == "torch":
            self.transport = TorchTransport(group)
            assert (self.transport.rank, self.transport.nranks) == (rank, nranks), "slab != torch.distributed rank"
            self._check(lqcd_set_comm(self.ctx, self.transport.ops))
        elif comm == "nccl":
            import torch.distributed as dist
            if nranks > 1:
                assert dist.is_initialized() and dist.get_world_size(group) == nranks and dist.get_rank(group) == rank
            if rank == 0:
                rc, nccl_id = lqcd_nccl_unique_id()
                if rc != LQCD_OK:
                    raise LqcdError(rc, lqcd_last_error(None))
            else:
                nccl_id = None
            if nranks > 1:
                box = [nccl_id]
                dist.broadcast_object_list(box, src=dist.get_global_rank(group, 0) if group is not None else 0,
                                           group=group)
                nccl_id = box[0]
            self._check(lqcd_comm_init_nccl(self.ctx, nccl_id))
        elif comm == "p2p":
            import torch.distributed as dist
            rc, mine = lqcd_p2p_export(self.ctx)
            self._check(rc)
            handles = [mine]
            if nranks > 1:
                assert dist.is_initialized() and dist.get_world_size(group) == nranks and dist.get_rank(group) == rank
                handles = [None] * nranks
                dist.all_gather_object(handles, mine, group=group)
            self._check(lqcd_comm_init_p2p(self.ctx, b"".join(handles)))
        else:
            raise ValueError(f"unknown transport {comm!r}")

    # -- slab bookkeeping (slicing only): the part of a whole-lattice tensor this rank owns.  The cut is along t,
    # the slowest index, so a slab is one contiguous range of sites.
    @staticmethod
    def slab_range(L_global: Sequence[int], rank: int, nranks: int):
        """(first, last+1) lexicographic site index of the slab."""
        v3 = int(L_global[0]) * int(L_global[1]) * int(L_global[2])
        lt = int(L_global[3]) // nranks
        return rank * lt * v3, (rank + 1) * lt * v3

    @staticmethod
    def slab_of_links(links, L_global, rank, nranks):
        """(4, V, 3, 3, 2) -> (4, V_local, 3, 3, 2), contiguous"""
        a, b = Lattice.slab_range(L_global, rank, nranks)
        return links[:, a:b].contiguous()

    @staticmethod
    def slab_of_vector(v, L_global, rank, nranks):
        """parity vector (3, Vh, 2) -> (3, Vh_local, 2), contiguous"""
        a, b = Lattice.slab_range(L_global, rank, nranks)
        return v[:, a // 2:b // 2].contiguous()

    def close(self):
        if getattr(self, "ctx", None):
            lqcd_destroy(self.ctx)
            self.ctx = None

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass

    # -- helpers
    def _check(self, rc: int, allow=()):
        if rc != LQCD_OK and rc not in allow:
            raise LqcdError(rc, lqcd_last_error(self.ctx))
        return rc

    def _sync_stream(self):
        self._check(lqcd_set_stream(self.ctx, self._torch.cuda.current_stream().cuda_stream))

    def _t(self, t, shape, device_type=None, dtype=None):
        torch = self._torch
        dtype = torch.float64 if dtype is None else dtype
        assert t.dtype == dtype and t.is_contiguous(), f"{dtype} contiguous tensor expected"
        assert tuple(t.shape) == tuple(shape), f"shape {tuple(t.shape)} != {tuple(shape)}"
        if device_type is not None:
            assert t.device.type == device_type
        return t.data_ptr()

    def _f32(self, t) -> bool:
        torch = self._torch
        assert t.dtype in (torch.float64, torch.float32), "float64 or float32 tensor expected"
        return t.dtype == torch.float32

    def new_vector(self, n: Optional[int] = None, dtype=None):
        shape = (3, self.Vh, 2) if n is None else (n, 3, self.Vh, 2)
        return self._torch.empty(shape, dtype=dtype or self._torch.float64, device="cuda")

    # -- options / stats
    def set_option(self, key, value):
        self._check(lqcd_set_option(self.ctx, key, value))

    def get_option(self, key) -> float:
        rc, v = lqcd_get_option(self.ctx, key)
        self._check(rc)
        return v

    def stat(self, key, idx=0) -> float:
        rc, v = lqcd_get_stat(self.ctx, key, idx)
        self._check(rc)
        return v

    @property
    def launches(self) -> int:
        return int(self.stat(LQCD_STAT_GPU_LAUNCHES))

    # -- the path
    def set_gauge(self, links):
        """links: (4, V, 3, 3, 2) float64, canonical layout; CUDA or CPU tensor."""
        p = self._t(links, (4, self.V, 3, 3, 2))
        self._sync_stream()
        if links.device.type == "cuda":
            self._check(lqcd_set_gauge(self.ctx, p))
        else:
            self._check(lqcd_set_gauge_host(self.ctx, p))

    def set_u1_phases(self, theta):
        """theta: (4, V) float64 angles of u_mu(x) = exp(i theta_mu(x)), CUDA or CPU tensor;
        None switches the field off."""
        self._sync_stream()
        if theta is None:
            self._check(lqcd_set_u1_phases(self.ctx, None))
            return
        p = self._t(theta, (4, self.V))
        if theta.device.type == "cuda":
            self._check(lqcd_set_u1_phases(self.ctx, p))
        else:
            self._check(lqcd_set_u1_phases_host(self.ctx, p))

    def _apply(self, fns, v, out):
        torch = self._torch
        f32 = self._f32(v)
        pin = self._t(v, (3, self.Vh, 2), dtype=v.dtype)
        if out is None:
            out = torch.empty_like(v)
        pout = self._t(out, (3, self.Vh, 2), v.device.type, v.dtype)
        self._sync_stream()
        self._check(fns[2 * f32 + (v.device.type != "cuda")](self.ctx, pout, pin))
        return out

    def doe(self, v_even, out=None):
        """D_oe: even -> odd parity vector."""
        return self._apply((lqcd_doe, lqcd_doe_host, lqcd_doe_f32, lqcd_doe_f32_host), v_even, out)

    def deo(self, v_odd, out=None):
        """D_eo: odd -> even parity vector."""
        return self._apply((lqcd_deo, lqcd_deo_host, lqcd_deo_f32, lqcd_deo_f32_host), v_odd, out)

    def mdagm(self, v_even, sigma: float = 0.0, out=None):
        """(m^2 + sigma) v - D_eo D_oe v."""
        f32 = self._f32(v_even)
        pin = self._t(v_even, (3, self.Vh, 2), "cuda", v_even.dtype)
        if out is None:
            out = self._torch.empty_like(v_even)
        pout = self._t(out, (3, self.Vh, 2), "cuda", v_even.dtype)
        self._sync_stream()
        self._check((lqcd_mdagm_f32 if f32 else lqcd_mdagm)(self.ctx, pout, pin, sigma))
        return out

    def comm_abort(self):
        """This rank cannot go on: release the ranks that wait for it (include/lqcd.h, lqcd_comm_abort)."""
        self._check(lqcd_comm_abort(self.ctx))

    def mdagm_static(self, v_even, out, sigma: float = 0.0):
        """``mdagm`` through ``lqcd_mdagm_static``: for callers that cannot allocate device memory (their application
        owns all of it, or they must not trigger the device-wide synchronisation of cudaMalloc).  ``out`` is
        therefore required, double precision only, at most ``LQCD_STATIC_MAX_VH`` sites per parity; the temporary
        sits in a 3 MiB buffer built into the library and shared by every caller on the device, so calls must not
        overlap on the GPU (include/lqcd.h)."""
        pin = self._t(v_even, (3, self.Vh, 2), "cuda", self._torch.float64)
        pout = self._t(out, (3, self.Vh, 2), "cuda", self._torch.float64)
        self._sync_stream()
        self._check(lqcd_mdagm_static(self.ctx, pout, pin, sigma))
        return out

    def mshift_cg(self, b_even, shifts: Sequence[float], tol: float, x=None, raise_on_noconv: bool = True):
        """Solve (m^2 - D_eo D_oe + shifts[i]) x[i] = b.  Returns (x, info); x is (nshift, 3, Vh, 2)."""
        torch = self._torch
        n = len(shifts)
        f32 = self._f32(b_even)
        pb = self._t(b_even, (3, self.Vh, 2), dtype=b_even.dtype)
        if x is None:
            x = torch.empty((n, 3, self.Vh, 2), dtype=b_even.dtype, device=b_even.device,
                            pin_memory=(b_even.device.type == "cpu"))
        self._t(x, (n, 3, self.Vh, 2), b_even.device.type, b_even.dtype)
        ptrs = [x[i].data_ptr() for i in range(n)]
        self._sync_stream()
        fn = (lqcd_mshift_cg, lqcd_mshift_cg_host, lqcd_mshift_cg_f32, lqcd_mshift_cg_f32_host)[
            2 * f32 + (b_even.device.type != "cuda")]
        rc = fn(self.ctx, pb, shifts, tol, ptrs)
        self._check(rc, allow=() if raise_on_noconv else (LQCD_ENOCONV,))
        return x, self._solve_info(rc, n)

    def mshift_cg_mixed(self, b_even, shifts: Sequence[float], tol: float, x=None, raise_on_noconv: bool = True):
        """The same systems to a double-precision tolerance on the TRUE residual, iterating in single precision with
        double-precision reliable updates (include/lqcd.h: lqcd_mshift_cg_mixed).  float64 CUDA tensors."""
        torch = self._torch
        n = len(shifts)
        pb = self._t(b_even, (3, self.Vh, 2), "cuda")
        if x is None:
            x = torch.empty((n, 3, self.Vh, 2), dtype=torch.float64, device="cuda")
        self._t(x, (n, 3, self.Vh, 2), "cuda")
        self._sync_stream()
        rc = lqcd_mshift_cg_mixed(self.ctx, pb, shifts, tol, [x[i].data_ptr() for i in range(n)])
        self._check(rc, allow=() if raise_on_noconv else (LQCD_ENOCONV,))
        info = self._solve_info(rc, n)
        info["reliable_updates"] = int(self.stat(LQCD_STAT_RELIABLE_UPDATES))
        return x, info

    def _solve_info(self, rc, n):
        return dict(
            status=rc,
            iters=int(self.stat(LQCD_STAT_ITERS)),
            rel_res=self.stat(LQCD_STAT_REL_RES),
            freeze_iter=[int(self.stat(LQCD_STAT_FREEZE_ITER, i)) for i in range(n)],
            base_shift=int(self.stat(LQCD_STAT_BASE_SHIFT)),
            solve_ms=self.stat(LQCD_STAT_SOLVE_MS),
            graph_replays=int(self.stat(LQCD_STAT_GRAPH_REPLAYS)),
            solver_path=int(self.stat(LQCD_STAT_SOLVER_PATH)),
        )

    def rational_apply(self, b_even, alpha0: float, alpha: Sequence[float], shifts: Sequence[float], tol: float,
                       y=None, raise_on_noconv: bool = True):
        """y = alpha0 b + sum_i alpha_i (m^2 - D_eo D_oe + shifts[i])^-1 b, accumulated
        during the multi-shift solve.  Returns (y, info)."""
        torch = self._torch
        f32 = self._f32(b_even)
        pb = self._t(b_even, (3, self.Vh, 2), dtype=b_even.dtype)
        host = b_even.device.type == "cpu"
        assert not (f32 and host), "no host entry point for the single-precision rational sum"
        if y is None:
            y = torch.empty((3, self.Vh, 2), dtype=b_even.dtype, device=b_even.device, pin_memory=host)
        py = self._t(y, (3, self.Vh, 2), b_even.device.type, b_even.dtype)
        self._sync_stream()
        if f32:
            rc = lqcd_rational_apply_f32(self.ctx, pb, alpha0, alpha, shifts, tol, py)
        else:
            rc = lqcd_rational_apply(self.ctx, pb, alpha0, alpha, shifts, tol, py, host=host)
        self._check(rc, allow=() if raise_on_noconv else (LQCD_ENOCONV,))
        return y, self._solve_info(rc, len(shifts))

    def pack(self, site_field, parity: int, out=None):
        """(V,3,2) site field -> (3,Vh,2) parity vector of the given parity."""
        f32 = self._f32(site_field)
        ps = self._t(site_field, (self.V, 3, 2), "cuda", site_field.dtype)
        if out is None:
            out = self.new_vector(dtype=site_field.dtype)
        self._sync_stream()
        fn = lqcd_pack_vector_f32 if f32 else lqcd_pack_vector
        self._check(fn(self.ctx, parity, ps, self._t(out, (3, self.Vh, 2), "cuda", site_field.dtype)))
        return out

    def unpack(self, v, parity: int, out=None):
        """(3,Vh,2) parity vector -> (V,3,2) site field (other parity zero unless `out` is given)."""
        f32 = self._f32(v)
        pv = self._t(v, (3, self.Vh, 2), "cuda", v.dtype)
        if out is None:
            out = self._torch.zeros((self.V, 3, 2), dtype=v.dtype, device="cuda")
        self._sync_stream()
        fn = lqcd_unpack_vector_f32 if f32 else lqcd_unpack_vector
        self._check(fn(self.ctx, parity, pv, self._t(out, (self.V, 3, 2), "cuda", v.dtype)))
        return out
