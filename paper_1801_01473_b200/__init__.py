"""paper_1801_01473_b200 -- B200 staggered Dslash + multi-shift CG (arxiv/paper_1801_01473 hot path).

Thin ctypes binding over the C ABI of ``include/lqcd.h`` (``liblqcd_b200.so``, built in tree by
``python -m paper_1801_01473_b200.build``).  Argument marshalling only: every step of the path runs in
the CUDA kernels under ``csrc/``.  There is no CPU fallback -- if the library is missing or no GPU is
present the calls raise.

Functions carry the C names (``lqcd_create`` ...); :class:`Lattice` is a small convenience wrapper that
takes torch tensors (device memory and streams are torch's job, nothing else is).
"""
from .binding import (  # noqa: F401
    LQCD_OK, LQCD_EINVAL, LQCD_ENOGAUGE, LQCD_ENOMEM, LQCD_ECUDA, LQCD_ENOCONV, LQCD_EBREAKDOWN, LQCD_ENOTSU3, LQCD_ECOMM, LQCD_NCCL_ID_BYTES, LQCD_P2P_HANDLE_BYTES,
    LQCD_OPT_MASS, LQCD_OPT_ANTIPERIODIC_T, LQCD_OPT_RECON, LQCD_OPT_MAX_ITER, LQCD_OPT_CHECK_EVERY,
    LQCD_OPT_USE_GRAPH, LQCD_OPT_LINK_PRECISIONS, LQCD_OPT_SHIFT_BLOCK, LQCD_OPT_PERSISTENT, LQCD_PREC_F64, LQCD_PREC_F32,
    LQCD_STAT_ITERS, LQCD_STAT_REL_RES, LQCD_STAT_FREEZE_ITER, LQCD_STAT_BASE_SHIFT, LQCD_STAT_GPU_LAUNCHES,
    LQCD_STAT_SOLVE_MS, LQCD_STAT_RELIABLE_UPDATES, LQCD_STAT_GRAPH_REPLAYS, LQCD_STAT_SOLVER_PATH,
    LqcdError, Lattice, load_library, library_path, EXPORTS,
    lqcd_create, lqcd_destroy, lqcd_set_stream, lqcd_set_option, lqcd_get_option, lqcd_workspace_bytes,
    lqcd_set_workspace, lqcd_set_gauge, lqcd_set_gauge_host, lqcd_set_u1_phases, lqcd_set_u1_phases_host, lqcd_doe, lqcd_deo, lqcd_doe_host, lqcd_deo_host,
    lqcd_mdagm, lqcd_mshift_cg, lqcd_mshift_cg_host, lqcd_rational_apply, lqcd_rational_apply_host, lqcd_get_stat, lqcd_pack_vector, lqcd_unpack_vector,
    lqcd_last_error,
    lqcd_doe_f32, lqcd_deo_f32, lqcd_doe_f32_host, lqcd_deo_f32_host, lqcd_mdagm_f32, lqcd_mshift_cg_f32,
    lqcd_mshift_cg_f32_host, lqcd_rational_apply_f32, lqcd_pack_vector_f32, lqcd_unpack_vector_f32,
    lqcd_create_slab, lqcd_set_comm, lqcd_nccl_unique_id, lqcd_comm_init_nccl, lqcd_p2p_export, lqcd_comm_init_p2p, lqcd_slab_info, lqcd_comm_ops,
    TorchTransport, lqcd_mshift_cg_mixed, lqcd_mdagm_static, LQCD_STATIC_MAX_VH, lqcd_comm_abort, LQCD_OPT_COMM_TIMEOUT,
)
