// lqcd_api.cu -- the C ABI of include/lqcd.h: context, memory, gauge storage, operators, solver driver.
// Every step of the path runs in the kernels of dslash.cuh / cg.cuh; this file only validates
// arguments, owns device memory and enqueues launches.  There is no CPU fallback: without a CUDA
// device lqcd_create fails.
#include "../../include/lqcd.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <chrono>
#include <cstring>
#include <mutex>
#include <new>
#include <thread>
#include <vector>

#include "cg.cuh"
#include "comm.h"
#include "dslash.cuh"
#include "lqcd_internal.cuh"
#include "p2p.cuh"
#include "persist.cuh"

namespace {

thread_local char g_create_error[256] = "";

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t b) { return (b + ALIGN - 1) / ALIGN * ALIGN; }

#ifndef SLAB_GRAPH_MAX_VH
#define SLAB_GRAPH_MAX_VH (1u << 18)      // local sites per parity up to which a slab's CG iteration is replayed from a graph
#endif

#ifndef LINKS_RESIDENT_MAX
#define LINKS_RESIDENT_MAX (48u << 20)
#endif

}  // namespace

// everything that exists once per precision T (double: the default path; float: the *_f32 entry points)
template <typename T>
struct PrecBufs {
    V2<T>* W = nullptr;      // stored links
    size_t W_bytes = 0;
    int recon_stored = 0;    // 0 = no gauge in this precision, else 18 or 12
    T* Th = nullptr;         // stored U(1) angles theta_mu(x) (lqcd_set_u1_phases), [(mu*2+par)*Vh + k]
    int u1_stored = 0;
    V2<T> *p = nullptr, *t = nullptr;
    V2<T>* p_keep = nullptr;                 // p of the first iteration of the current block (CgState::p_keep)
    V2<T>* hist[LQCD_MAX_BLOCK] = {};        // ring of residual vectors (cg.cuh)
    int n_hist = 0;
    V2<T>* pextra[LQCD_MAX_SHIFTS] = {};
    int n_pextra = 0;
    cudaGraphExec_t graph_exec = nullptr;    // CUDA graph of `graph_iters` CG iterations
    int graph_iters = 0, graph_rational = 0, graph_block = 0;
    int graph_launches = 0;                  // kernels one replay of the graph launches
    // slab mode: faces of the input vector, [lo|hi][c][face] each; t-links leaving the slice below the slab
    V2<T>* halo_send = nullptr;
    V2<T>* halo_recv = nullptr;
    V2<T>* Wt_lo = nullptr;                  // [parity of origin][e][face]
    V2<T>* Wt_send = nullptr;                // one-time staging of my top t-links (+ a dummy receive buffer behind it)
    T* Th_lo = nullptr;                      // U(1) angles of those links, [parity of origin][face]
    T* Th_send = nullptr;
    V2<T>* stage_b = nullptr;                // host-call staging (device copies of host arguments)
    V2<T>* stage_x[LQCD_MAX_SHIFTS] = {};
    int n_stage_x = 0;
};

struct lqcd_ctx {
    int L[4];
    Geom g;
    size_t V, Vh;
    int device, num_sms;
    int coop_launch;         // the device supports cooperative launches (the persistent solver needs one)
    cudaStream_t stream;

    // options
    double mass;
    int recon_opt, max_iter, check_every, use_graph;
    int shift_block_opt;     // LQCD_OPT_SHIFT_BLOCK: 0 = chosen from the lattice size (block_len())
    int persistent_opt;      // LQCD_OPT_PERSISTENT: -1 = the library decides (lattices that live in L2), 0 = never, 1 = always
    double comm_timeout;     // LQCD_OPT_COMM_TIMEOUT, seconds; <= 0: wait for ever

    // memory
    char* arena;             // caller workspace (not owned) or NULL
    size_t arena_bytes, arena_used;
    std::vector<void*> owned;    // cudaMalloc'ed by us

    // stored gauge field, operator / solver buffers, CG graph and host-call staging: one set per precision
    PrecBufs<double> d;
    PrecBufs<float> f;
    int prec_opt;            // LQCD_OPT_LINK_PRECISIONS: which of them the next lqcd_set_gauge stores
    int u1_on;               // general U(1) phases in force (lqcd_set_u1_phases with a non-NULL field)
    double* dev_max;

    // slab decomposition (lqcd_create_slab): rank of nranks along t, transport, its stream and events
    int slab, rank, nranks;
    lqcd_comm_ops comm;
    bool has_comm;
    lqcd_nccl::Transport nccl;
    lqcd_p2p::Transport p2p;     // peer-memory transport (lqcd_comm_init_p2p)
    cudaStream_t comm_stream;
    cudaEvent_t ev_pack, ev_halo;
    double* red;             // device: the scalar product being reduced over ranks
    char* host_stage;        // pinned: staging of a host_staged transport (4 faces, or the link faces)
    size_t host_stage_bytes;
    double* red_host;        // pinned

    double* partials;
    size_t n_partials;
    CgState* st_dev;
    CgState* st_host;        // pinned
    int* flag_host;          // pinned, 2 ints
    double* max_host;        // pinned
    cudaEvent_t ev[2], ev_t0, ev_t1, ev_m0, ev_m1;
    bool basics;

    // statistics
    int last_iters, last_i0, last_nshift;
    double last_rel;
    int last_freeze[LQCD_MAX_SHIFTS];
    float last_ms;
    int last_updates;        // reliable updates of the last mixed-precision solve
    int last_replays;        // CUDA-graph replays of the last solve (0: launched plainly, or the persistent kernel)
    int last_path;           // LQCD_STAT_SOLVER_PATH of the last solve
    long long launches;

    char err[256];
};

namespace {

int fail(lqcd_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

#define CU(expr)                                                                                     \
    do {                                                                                             \
        cudaError_t e_ = (expr);                                                                     \
        if (e_ != cudaSuccess)                                                                       \
            return fail(c, LQCD_ECUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

int dev_alloc(lqcd_ctx* c, void** out, size_t bytes) {
    bytes = align_up(bytes);
    if (c->arena) {
        if (c->arena_used + bytes > c->arena_bytes)
            return fail(c, LQCD_ENOMEM, "workspace too small: need %zu more bytes", c->arena_used + bytes - c->arena_bytes);
        *out = c->arena + c->arena_used;
        c->arena_used += bytes;
        return LQCD_OK;
    }
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(c, LQCD_ENOMEM, "cudaMalloc(%zu) failed: %s", bytes, cudaGetErrorString(e));
    }
    c->owned.push_back(p);
    *out = p;
    return LQCD_OK;
}

// memory outside the caller's arena even when there is one: the staging copies of the *_host entry points
// (lqcd_workspace_bytes does not count them)
int dev_alloc_own(lqcd_ctx* c, void** out, size_t bytes) {
    char* arena = c->arena;
    c->arena = nullptr;
    const int rc = dev_alloc(c, out, bytes);
    c->arena = arena;
    return rc;
}

void dev_free_owned(lqcd_ctx* c, void* p) {
    for (size_t i = 0; i < c->owned.size(); ++i)
        if (c->owned[i] == p) {
            cudaFree(p);
            c->owned.erase(c->owned.begin() + i);
            return;
        }
}

template <typename T> const PrecBufs<T>& bufs_c(const lqcd_ctx* c);
template <> const PrecBufs<double>& bufs_c<double>(const lqcd_ctx* c) { return c->d; }
template <> const PrecBufs<float>& bufs_c<float>(const lqcd_ctx* c) { return c->f; }
template <typename T> PrecBufs<T>& bufs(lqcd_ctx* c);
template <> PrecBufs<double>& bufs<double>(lqcd_ctx* c) { return c->d; }
template <> PrecBufs<float>& bufs<float>(lqcd_ctx* c) { return c->f; }

template <typename T>
void drop_graph(lqcd_ctx* c) {
    PrecBufs<T>& B = bufs<T>(c);
    if (B.graph_exec) {
        cudaGraphExecDestroy(B.graph_exec);
        B.graph_exec = nullptr;
    }
    B.graph_iters = 0;
}
void drop_graphs(lqcd_ctx* c) {
    drop_graph<double>(c);
    drop_graph<float>(c);
}

// Block length m of the deferred shift updates (cg.cuh).  Default: 32 -- the longer the block, the fewer bytes per
// iteration (48 + 192 (n_act-1)/m + 144/m per site) -- except on lattices small enough to live in L2, which get 16,
// the longest block the persistent solver handles (persist.cuh).
int block_len(const lqcd_ctx* c) {
    if (c->shift_block_opt) return c->shift_block_opt;
    const size_t smallest_links = (size_t)8 * 6 * c->Vh * sizeof(float2);          // float, two rows
    return smallest_links <= LINKS_RESIDENT_MAX ? 16 : 32;
}

template <typename T> size_t vec_bytes(const lqcd_ctx* c) { return c->Vh * 3 * sizeof(V2<T>); }
template <typename T> size_t links_bytes(const lqcd_ctx* c, int recon) {
    return (size_t)8 * (recon == 12 ? 6 : 9) * c->Vh * sizeof(V2<T>);
}

// The stored links of precision T fit in L2 beside the solver's vectors (B200: 126 MB in two halves, and a line
// read by SMs of both dies may sit in both).  Measured at 16^4 (37.7 MB of links): with the streaming policy every
// application re-read them from DRAM (40 MB per launch under ncu --cache-control none); kept, one application in a
// graph takes 4.5 us = 9.6 TB/s out of L2.
template <typename T> int links_resident(const lqcd_ctx* c) {
    const int ne = (bufs_c<T>(c).recon_stored == 12) ? 6 : 9;
    return (size_t)8 * ne * c->Vh * sizeof(V2<T>) <= LINKS_RESIDENT_MAX ? 1 : 0;
}

// L2 eviction priorities of the operator's loads (dslash.cuh, l2_policy codes).  Neighbour vectors are re-used by 8
// sites: last to go.  Links: streamed once per application, first to go -- unless the whole stored field is small
// enough to stay in L2 for the next application (links_resident), where they too are last to go.  Measured at 16^4,
// whole CG iteration: links evict_first 36 us, evict_normal or evict_last 19 us, whatever the vectors' priority;
// pinning the links with a persisting access-policy window on the stream (40 or 79 MB set aside) changed nothing.
template <typename T> void set_policies(const lqcd_ctx* c, DslashArgs<T>& a) {
    a.pol_links = links_resident<T>(c) ? 2 : 0;
    a.pol_vecs = 2;
}

int ds_grid(const lqcd_ctx* c) { return (int)((c->Vh + DS_BLOCK - 1) / DS_BLOCK); }
int cg_grid(const lqcd_ctx* c) {
    const size_t n = c->Vh * 3;
    size_t blocks = (n + CG_BLOCK - 1) / CG_BLOCK;
    const size_t cap = (size_t)c->num_sms * 8;
    return (int)(blocks < cap ? blocks : cap);
}

// one partial per block of the largest launch; the persistent solver keeps two arrays of its grid
size_t n_partials_needed(const lqcd_ctx* c) {
    size_t n = (size_t)(ds_grid(c) > cg_grid(c) ? ds_grid(c) : cg_grid(c));
    const size_t resident = (size_t)c->num_sms * 16;       // no kernel of the library has more blocks per SM than this
    if (n < resident) n = resident;
    return 2 * n + 8;
}

// buffers every call needs: the CG state, reduction partials, pinned mirrors, events
int ensure_basics(lqcd_ctx* c) {
    if (c->basics) return LQCD_OK;
    // every resource is created only if it does not exist yet: a call that failed half way can be repeated
    int rc;
    if (!c->st_dev) {
        if ((rc = dev_alloc(c, (void**)&c->st_dev, sizeof(CgState)))) return rc;
        CU(cudaMemsetAsync(c->st_dev, 0, sizeof(CgState), c->stream));
    }
    if (!c->partials) {
        c->n_partials = n_partials_needed(c);
        if ((rc = dev_alloc(c, (void**)&c->partials, c->n_partials * sizeof(double)))) return rc;
    }
    if (!c->red && (rc = dev_alloc(c, (void**)&c->red, 2 * sizeof(double)))) return rc;
    if (!c->red_host) CU(cudaMallocHost((void**)&c->red_host, 2 * sizeof(double)));
    if (c->slab) {
        if (!c->comm_stream) {
            // highest priority: the blocks of the border launch are few and should not queue behind what is left of
            // the interior launch (20,000 blocks at 48^4), or they become a tail of their own
            int lo = 0, hi = 0;
            CU(cudaDeviceGetStreamPriorityRange(&lo, &hi));
            CU(cudaStreamCreateWithPriority(&c->comm_stream, cudaStreamNonBlocking, hi));
        }
        if (!c->ev_pack) CU(cudaEventCreateWithFlags(&c->ev_pack, cudaEventDisableTiming));
        if (!c->ev_halo) CU(cudaEventCreateWithFlags(&c->ev_halo, cudaEventDisableTiming));
    }
    if (!c->dev_max && (rc = dev_alloc(c, (void**)&c->dev_max, sizeof(double)))) return rc;
    if (!c->st_host) CU(cudaMallocHost((void**)&c->st_host, sizeof(CgState)));
    if (!c->flag_host) CU(cudaMallocHost((void**)&c->flag_host, 2 * sizeof(int)));
    if (!c->max_host) CU(cudaMallocHost((void**)&c->max_host, sizeof(double)));
    for (int i = 0; i < 2; ++i)
        if (!c->ev[i]) CU(cudaEventCreateWithFlags(&c->ev[i], cudaEventDisableTiming));
    if (!c->ev_t0) CU(cudaEventCreate(&c->ev_t0));
    if (!c->ev_t1) CU(cudaEventCreate(&c->ev_t1));
    if (!c->ev_m0) CU(cudaEventCreate(&c->ev_m0));
    if (!c->ev_m1) CU(cudaEventCreate(&c->ev_m1));
    c->basics = true;
    return LQCD_OK;
}

// the odd-parity temporary of the two-launch operators
template <typename T>
int ensure_tmp(lqcd_ctx* c) {
    int rc;
    if ((rc = ensure_basics(c))) return rc;
    PrecBufs<T>& B = bufs<T>(c);
    if (!B.t && (rc = dev_alloc(c, (void**)&B.t, vec_bytes<T>(c)))) return rc;
    return LQCD_OK;
}

template <typename T>
int ensure_solver(lqcd_ctx* c, int nshift) {
    int rc;
    if ((rc = ensure_tmp<T>(c))) return rc;
    PrecBufs<T>& B = bufs<T>(c);
    while (B.n_hist < block_len(c)) {
        if ((rc = dev_alloc(c, (void**)&B.hist[B.n_hist], vec_bytes<T>(c)))) return rc;
        ++B.n_hist;
    }
    if (!B.p && (rc = dev_alloc(c, (void**)&B.p, vec_bytes<T>(c)))) return rc;
    if (!B.p_keep && (rc = dev_alloc(c, (void**)&B.p_keep, vec_bytes<T>(c)))) return rc;
    while (B.n_pextra < nshift - 1) {
        if ((rc = dev_alloc(c, (void**)&B.pextra[B.n_pextra], vec_bytes<T>(c)))) return rc;
        ++B.n_pextra;
    }
    return LQCD_OK;
}

template <typename T, int EPI, int U1>
void launch_dslash_u(lqcd_ctx* c, const DslashArgs<T>& a) {
    if (bufs<T>(c).recon_stored == 12)
        dslash_kernel<T, 12, EPI, U1><<<ds_grid(c), DS_BLOCK, 0, c->stream>>>(a);
    else
        dslash_kernel<T, 18, EPI, U1><<<ds_grid(c), DS_BLOCK, 0, c->stream>>>(a);
    ++c->launches;
}
template <typename T, int EPI>
void launch_dslash_t(lqcd_ctx* c, const DslashArgs<T>& a) {
    if (c->u1_on) launch_dslash_u<T, EPI, 1>(c, a);
    else launch_dslash_u<T, EPI, 0>(c, a);
}

// ---- slab mode ------------------------------------------------------------------------------------------------
#define COMM(expr)                                                                                   \
    do {                                                                                             \
        if ((expr) != 0) return fail(c, LQCD_ECOMM, "transport failed in %s (%s:%d)", #expr, __FILE__, __LINE__); \
    } while (0)

size_t face_sites(const lqcd_ctx* c) { return (size_t)c->g.st; }

int ensure_host_stage(lqcd_ctx* c, size_t bytes) {
    if (c->host_stage_bytes >= bytes) return LQCD_OK;
    if (c->host_stage) cudaFreeHost(c->host_stage);
    c->host_stage = nullptr;
    c->host_stage_bytes = 0;
    CU(cudaMallocHost((void**)&c->host_stage, bytes));
    c->host_stage_bytes = bytes;
    return LQCD_OK;
}

// ring exchange of two device buffers of `bytes` each, ordered after the work enqueued on c->comm_stream
int comm_exchange(lqcd_ctx* c, const void* send_lo, const void* send_hi, void* recv_lo, void* recv_hi, size_t bytes) {
    if (!c->comm.host_staged) {
        COMM(c->comm.exchange(c->comm.user, send_lo, send_hi, recv_lo, recv_hi, bytes, (void*)c->comm_stream));
        return LQCD_OK;
    }
    int rc;
    if ((rc = ensure_host_stage(c, 4 * bytes))) return rc;
    char* h = c->host_stage;
    CU(cudaMemcpyAsync(h, send_lo, bytes, cudaMemcpyDeviceToHost, c->comm_stream));
    CU(cudaMemcpyAsync(h + bytes, send_hi, bytes, cudaMemcpyDeviceToHost, c->comm_stream));
    CU(cudaStreamSynchronize(c->comm_stream));
    COMM(c->comm.exchange(c->comm.user, h, h + bytes, h + 2 * bytes, h + 3 * bytes, bytes, nullptr));
    CU(cudaMemcpyAsync(recv_lo, h + 2 * bytes, bytes, cudaMemcpyHostToDevice, c->comm_stream));
    CU(cudaMemcpyAsync(recv_hi, h + 3 * bytes, bytes, cudaMemcpyHostToDevice, c->comm_stream));
    CU(cudaStreamSynchronize(c->comm_stream));       // the staging buffer is free again on return
    return LQCD_OK;
}

// c->red[0] <- sum over ranks, on the compute stream
int comm_allreduce(lqcd_ctx* c) {
    if (!c->comm.host_staged) {
        COMM(c->comm.allreduce_sum(c->comm.user, c->red, 1, (void*)c->stream));
        return LQCD_OK;
    }
    CU(cudaMemcpyAsync(c->red_host, c->red, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    COMM(c->comm.allreduce_sum(c->comm.user, c->red_host, 1, nullptr));
    CU(cudaMemcpyAsync(c->red, c->red_host, sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CU(cudaStreamSynchronize(c->stream));            // red_host may be rewritten by the next reduction
    return LQCD_OK;
}

template <typename T>
int ensure_halo(lqcd_ctx* c) {
    int rc;
    PrecBufs<T>& B = bufs<T>(c);
    const size_t fb = 2 * 3 * face_sites(c) * sizeof(V2<T>);
    if (!B.halo_send && (rc = dev_alloc(c, (void**)&B.halo_send, fb))) return rc;
    if (!B.halo_recv && (rc = dev_alloc(c, (void**)&B.halo_recv, fb))) return rc;
    return LQCD_OK;
}

// SLAB = 2: the interior launch (no hop leaves the slab); SLAB = 1: the border slices (halo buffers on the t-hops)
template <typename T, int EPI, int U1, int SLAB>
void launch_dslash_slab_u(lqcd_ctx* c, const DslashArgs<T>& a, int grid, cudaStream_t stream) {
    if (bufs<T>(c).recon_stored == 12)
        dslash_kernel<T, 12, EPI, U1, SLAB><<<grid, DS_BLOCK, 0, stream>>>(a);
    else
        dslash_kernel<T, 18, EPI, U1, SLAB><<<grid, DS_BLOCK, 0, stream>>>(a);
    ++c->launches;
}
template <typename T, int EPI>
void launch_dslash_slab_k(lqcd_ctx* c, const DslashArgs<T>& a, int grid, cudaStream_t stream, bool interior) {
    if (interior) {
        if (c->u1_on) launch_dslash_slab_u<T, EPI, 1, 2>(c, a, grid, stream);
        else launch_dslash_slab_u<T, EPI, 0, 2>(c, a, grid, stream);
    } else {
        if (c->u1_on) launch_dslash_slab_u<T, EPI, 1, 1>(c, a, grid, stream);
        else launch_dslash_slab_u<T, EPI, 0, 1>(c, a, grid, stream);
    }
}

// One operator sweep on a slab (Alg. 1 of the paper): the two faces of the input are packed and
// sent, the interior time slices are computed meanwhile, the two border slices once the halos have arrived.
// `a` carries everything but the slab fields; kepi is the kernel's EPI (0, 2: operators; 4, 5: the two launches of the
// fused CG iteration, which write block partials to c->partials[0 .. *n_part): slab_reduce_step follows).
// The faces that travel are those of `face_v`, or, with face_v2, of face_v + beta face_v2 (K1: p = r + beta p_old,
// formed by the owner of the sites).
template <typename T>
int slab_apply(lqcd_ctx* c, DslashArgs<T>& a, int kepi, const V2<T>* face_v, const V2<T>* face_v2, int* n_part) {
    int rc;
    if (!c->has_comm) return fail(c, LQCD_ECOMM, "slab context without a transport (lqcd_comm_init_nccl / lqcd_set_comm)");
    if ((rc = ensure_halo<T>(c))) return rc;
    PrecBufs<T>& B = bufs<T>(c);
    const size_t face = face_sites(c), vh = c->Vh;
    const size_t row = face * sizeof(V2<T>), pitch = vh * sizeof(V2<T>);
    V2<T>* send_lo = B.halo_send;
    V2<T>* send_hi = B.halo_send + 3 * face;
    V2<T>* recv_lo = B.halo_recv;
    V2<T>* recv_hi = B.halo_recv + 3 * face;
    // peer-memory transport: the faces are written straight into the neighbours' halo buffers (no send buffer, no
    // transport kernel), and the border launch reads my halos where the neighbours wrote them (p2p.cuh)
    const bool p2p = c->p2p.active && c->comm.user == (void*)&c->p2p;
    if (p2p && c->p2p.dead) return fail(c, LQCD_ECOMM, "peer-memory transport has failed: %s", c->p2p.error);
    if (p2p) {
        const lqcd_p2p::Slots o = lqcd_p2p::begin(&c->p2p);
        send_lo = (V2<T>*)o.dst_dn;
        send_hi = (V2<T>*)o.dst_up;
        recv_lo = (V2<T>*)o.recv_lo;
        recv_hi = (V2<T>*)o.recv_hi;
    }
    // the input is complete at this point of the compute stream; everything about the faces happens on the
    // communication stream from here on, beside the interior launch
    CU(cudaEventRecord(c->ev_pack, c->stream));
    CU(cudaStreamWaitEvent(c->comm_stream, c->ev_pack, 0));
    if (face_v2) {
        slab_pack_p_kernel<T><<<(int)((6 * face + 255) / 256), 256, 0, c->comm_stream>>>(face_v, face_v2, send_lo, send_hi, c->st_dev, vh, face);
        ++c->launches;
    } else {
        // a face is three contiguous runs (one per colour) of the vector: strided copies, no kernel
        CU(cudaMemcpy2DAsync(send_lo, row, face_v, pitch, row, 3, cudaMemcpyDefault, c->comm_stream));
        CU(cudaMemcpy2DAsync(send_hi, row, face_v + (vh - face), pitch, row, 3, cudaMemcpyDefault, c->comm_stream));
    }

    a.g = c->g;
    a.W = B.W;
    set_policies<T>(c, a);
    a.Th = B.Th;
    a.Th_lo = B.Th_lo;
    a.partials = c->partials;
    a.st = c->st_dev;
    a.in_lo = recv_lo;
    a.in_hi = recv_hi;
    a.Wt_lo = B.Wt_lo;
    a.clear0 = a.clear1 = nullptr;      // set for the border launch only (peer-memory transport)
    // interior: t = 1 .. Lt-2; borders: t = 0 and t = Lt-1
    const int n_int = (int)(vh - 2 * face);
    const int grid_int = n_int > 0 ? (n_int + DS_BLOCK - 1) / DS_BLOCK : 0;
    const int grid_bor = (int)((2 * face + DS_BLOCK - 1) / DS_BLOCK);
    int part = 0;
    auto launch = [&](int grid, cudaStream_t stream, bool interior) {
        a.part_off = part;
        if (kepi == 0) launch_dslash_slab_k<T, 0>(c, a, grid, stream, interior);
        else if (kepi == 2) launch_dslash_slab_k<T, 2>(c, a, grid, stream, interior);
        else if (kepi == 4) launch_dslash_slab_k<T, 4>(c, a, grid, stream, interior);
        else launch_dslash_slab_k<T, 5>(c, a, grid, stream, interior);
        part += grid;
    };
    if (n_int > 0) {
        a.k0a = (int)face;
        a.na = n_int;
        a.k0b = 0;
        a.nsites = n_int;
        launch(grid_int, c->stream, true);
    }
    // faces in flight on the communication stream; the two border slices (t = 0 and t = Lt-1) follow them on
    // that stream, so they run beside the interior (disjoint outputs and partial slots) instead of after it
    if (p2p) {
        if (lqcd_p2p::signal_wait(&c->p2p, c->comm_stream, false)) return fail(c, LQCD_ECOMM, "peer-memory transport: %s", c->p2p.error);
        lqcd_p2p::clear_words(&c->p2p, &a.clear0, &a.clear1);
    } else if ((rc = comm_exchange(c, send_lo, send_hi, recv_lo, recv_hi, 3 * row))) {
        return rc;
    }
    a.k0a = 0;
    a.na = (int)face;
    a.k0b = (int)(vh - face);
    a.nsites = (int)(2 * face);
    launch(grid_bor, c->comm_stream, false);
    CU(cudaEventRecord(c->ev_halo, c->comm_stream));
    CU(cudaStreamWaitEvent(c->stream, c->ev_halo, 0));
    CU(cudaGetLastError());
    if (n_part) *n_part = part;
    return LQCD_OK;
}

// out(par) = D in on a slab, optionally with the epilogue out = coef pv - D in (epi == 2)
template <typename T>
int slab_dslash(lqcd_ctx* c, int epi, V2<T>* out, const V2<T>* in, int par, const V2<T>* pv, double coef) {
    DslashArgs<T> a{};
    a.in = in;
    a.out = out;
    a.par = par;
    a.pv = pv;
    a.coef = coef;
    return slab_apply<T>(c, a, epi, in, nullptr, nullptr);
}

// sum of c->partials[0..n) over this rank's blocks, then over the ranks, then the scalar step `which`.
// Peer-memory transport: the kernel that sums the partials stores the rank's sum into every rank's window itself, and
// the kernel of the scalar step adds the ranks' slots (two kernels and nranks stream waits per scalar product).
int slab_reduce_step(lqcd_ctx* c, int n, int which, double tol, int check_stop) {
    int rc;
    if (which != 0 && c->p2p.active && c->comm.user == (void*)&c->p2p) {
        lqcd_p2p::Transport* t = &c->p2p;
        if (t->dead) return fail(c, LQCD_ECOMM, "peer-memory transport has failed: %s", t->error);
        sum_partials_kernel<<<1, CG_BLOCK, 0, c->stream>>>(c->partials, n, c->red, c->st_dev, check_stop, lqcd_p2p::reduce_begin(t));
        if (lqcd_p2p::reduce_wait(t, c->stream)) return fail(c, LQCD_ECOMM, "peer-memory transport: %s", t->error);
        cg_scalar_slots_kernel<<<1, 64, 0, c->stream>>>(c->st_dev, lqcd_p2p::reduce_slots(t), lqcd_p2p::reduce_flags(t),
                                                        t->nranks, LQCD_P2P_RED_MAX, which);
    } else {
        sum_partials_kernel<<<1, CG_BLOCK, 0, c->stream>>>(c->partials, n, c->red, c->st_dev, check_stop, nullptr);
        if ((rc = comm_allreduce(c))) return rc;
        cg_scalar_kernel<<<1, 64, 0, c->stream>>>(c->st_dev, c->red, which, tol);
    }
    c->launches += 2;
    CU(cudaGetLastError());
    return LQCD_OK;
}

// out(par) = D in, optionally with the epilogue
template <typename T>
void launch_dslash(lqcd_ctx* c, int epi, V2<T>* out, const V2<T>* in, int par, const V2<T>* pv, double coef,
                   int check_stop) {
    DslashArgs<T> a{};
    a.g = c->g;
    a.W = bufs<T>(c).W;
    set_policies<T>(c, a);
    a.Th = bufs<T>(c).Th;
    a.in = in;
    a.out = out;
    a.par = par;
    a.pv = pv;
    a.coef = coef;
    a.partials = c->partials;
    a.st = c->st_dev;
    a.check_stop = check_stop;
    if (epi == 0) launch_dslash_t<T, 0>(c, a);
    else launch_dslash_t<T, 2>(c, a);
}

// after K1 (which = 1) / K2 (which = 2) of the whole-lattice path: block partials -> sum -> scalar step, one block
void launch_reduce_scalar(lqcd_ctx* c, int which, const double* partials) {
    cg_reduce_scalar_kernel<<<1, CG_BLOCK, 0, c->stream>>>(c->st_dev, partials, ds_grid(c), which);
    ++c->launches;
}

// Small whole lattices: the scalar step after a sweep rides in the NEXT sweep (dslash_kernel, FS = 1) instead of a
// one-block launch of its own, which is a third of the iteration there (16^4: 7.3 + 3.8 + 6.7 + 3.8 us).  Every block of
// the next sweep adds the partials itself, so their number must stay small.
#ifndef FS_MAX_BLOCKS
#define FS_MAX_BLOCKS 1024
#endif
bool fused_scalar(const lqcd_ctx* c) { return !c->slab && ds_grid(c) <= FS_MAX_BLOCKS; }
// K1 writes its partials to the first half of c->partials, K2 to the second (each is read while the other is written)
double* partials_k2(const lqcd_ctx* c) { return c->partials + (c->n_partials - 8) / 2; }

template <typename T, int EPI, int U1>
void launch_dslash_fs_u(lqcd_ctx* c, const DslashArgs<T>& a) {
    if (bufs<T>(c).recon_stored == 12)
        dslash_kernel<T, 12, EPI, U1, 0, 1><<<ds_grid(c) + 1, DS_BLOCK, 0, c->stream>>>(a);
    else
        dslash_kernel<T, 18, EPI, U1, 0, 1><<<ds_grid(c) + 1, DS_BLOCK, 0, c->stream>>>(a);
    ++c->launches;
}
template <typename T, int EPI>
void launch_dslash_fs(lqcd_ctx* c, const DslashArgs<T>& a) {
    if (c->u1_on) launch_dslash_fs_u<T, EPI, 1>(c, a);
    else launch_dslash_fs_u<T, EPI, 0>(c, a);
}

// The two launches of a fused CG iteration (dslash.cuh, EPI = 4 and 5; cg.cuh has the whole picture).
//   K1: t = D_oe p with p = r + beta p_old formed at the neighbours; <p,Ap>; a, zeta_i
//   K2: p, s = c0 p - D_eo t, r_new = r - a s, x_0 += a p at the thread's own site; |r_new|^2; beta, b_i, flags
template <typename T>
void launch_cg_fused(lqcd_ctx* c, const V2<T>* r_in, V2<T>* r_out, V2<T>* p_keep, int defer_base, int pos, int m) {
    PrecBufs<T>& B = bufs<T>(c);
    const bool fs = fused_scalar(c);
    DslashArgs<T> a{};
    a.g = c->g;
    a.W = B.W;
    set_policies<T>(c, a);
    a.Th = B.Th;
    a.partials = c->partials;
    a.st = c->st_dev;
    a.check_stop = 1;
    a.in = r_in;
    a.in2 = B.p;
    a.out = B.t;
    a.par = 1;
    if (fs) {
        // pos == 0: the step after K2 of the previous iteration was run by the launch that precedes the block sweep
        a.red_in = partials_k2(c);
        a.red_n = ds_grid(c);
        a.pending = (pos != 0);
        launch_dslash_fs<T, 4>(c, a);
    } else {
        launch_dslash_t<T, 4>(c, a);
        launch_reduce_scalar(c, 1, c->partials);
    }
    a.in = B.t;
    a.in2 = nullptr;
    a.out = nullptr;
    a.par = 0;
    a.pv = B.p;
    a.r_in = r_in;
    a.r_out = r_out;
    a.p_out = B.p;
    a.p_keep = p_keep;
    a.defer_base = defer_base;
    if (fs) {
        a.red_in = c->partials;
        a.partials = partials_k2(c);
        a.pending = 1;
        launch_dslash_fs<T, 5>(c, a);
        if (pos == m - 1) launch_reduce_scalar(c, 2, partials_k2(c));      // the block sweep needs the step done
    } else {
        launch_dslash_t<T, 5>(c, a);
        launch_reduce_scalar(c, 2, c->partials);
    }
}

// m >= 2: x_0 of the base system is updated by the block sweep too (CgState::defer_base)
int defer_base(const lqcd_ctx* c) { return block_len(c) >= 2 ? 1 : 0; }

// the sweep over the shifted systems that closes a block of iterations (K5 of cg.cuh)
template <typename T>
void launch_flush(lqcd_ctx* c) {
    const size_t n = c->Vh * 3;
    const int m = block_len(c);
    if (m <= 4) cg_flush_kernel<T, 4><<<cg_grid(c), CG_BLOCK, 0, c->stream>>>(c->st_dev, n);
    else if (m <= 8) cg_flush_kernel<T, 8><<<cg_grid(c), CG_BLOCK, 0, c->stream>>>(c->st_dev, n);
    else if (m <= 16) cg_flush_kernel<T, 16><<<cg_grid(c), CG_BLOCK, 0, c->stream>>>(c->st_dev, n);
    else cg_flush_kernel<T, 32><<<cg_grid(c), CG_BLOCK, 0, c->stream>>>(c->st_dev, n);
    ++c->launches;
}

// one CG iteration = K1, K2 (dslash.cuh), plus the block sweep when it is the last of a block; pos = iteration index mod m
template <typename T>
int launch_cg_iteration(lqcd_ctx* c, int pos) {
    const int m = block_len(c);
    PrecBufs<T>& B = bufs<T>(c);
    const int defer = defer_base(c);
    const V2<T>* r_in = B.hist[(pos + m - 1) % m];
    V2<T>* r_out = B.hist[pos];
    V2<T>* p_keep = (defer && pos == 0) ? B.p_keep : nullptr;
    if (c->slab) {
        // the same two launches with the two exchange steps of the slab decomposition: faces before each operator
        // sweep (of p, formed by its owner, before K1; of t before K2), one all-reduced double after each scalar
        // product, then the scalar step on every rank
        int rc, np = 0;
        DslashArgs<T> a{};
        a.check_stop = 1;
        a.in = r_in;
        a.in2 = B.p;
        a.out = B.t;
        a.par = 1;
        if ((rc = slab_apply<T>(c, a, 4, r_in, B.p, &np))) return rc;
        if ((rc = slab_reduce_step(c, np, 1, 0.0, 1))) return rc;
        a.in = B.t;
        a.in2 = nullptr;
        a.out = nullptr;
        a.par = 0;
        a.pv = B.p;
        a.r_in = r_in;
        a.r_out = r_out;
        a.p_out = B.p;
        a.p_keep = p_keep;
        a.defer_base = defer;
        if ((rc = slab_apply<T>(c, a, 5, B.t, nullptr, &np))) return rc;
        if ((rc = slab_reduce_step(c, np, 2, 0.0, 1))) return rc;
        if (pos == m - 1) launch_flush<T>(c);
        return LQCD_OK;
    }
    launch_cg_fused<T>(c, r_in, r_out, p_keep, defer, pos, m);
    if (pos == m - 1) launch_flush<T>(c);
    return LQCD_OK;
}

// ---- the whole solve as one cooperative kernel (persist.cuh) -----------------------------------------------------
template <typename T, int RECON, int U1>
int persistent_grid(const lqcd_ctx* c) {
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, cg_persistent_kernel<T, RECON, U1>, PS_BLOCK, 0) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    // every resident slot is used (the sites are dealt out evenly over the blocks, persist.cuh); one of the blocks
    // runs the scalar recurrences instead of sites; never more site blocks than sites
    const long cap = (long)per_sm * c->num_sms - 1;
    if (cap < 1) return 0;
    const long want = (long)((c->Vh + PS_BLOCK - 1) / PS_BLOCK);       // no more blocks than one site per thread needs
    return (int)(want < cap ? want : cap) + 1;
}

template <typename T, int RECON, int U1>
int launch_persistent_k(lqcd_ctx* c, PersistArgs<T>& P) {
    const int grid = persistent_grid<T, RECON, U1>(c);
    if (grid < 2) return fail(c, LQCD_ECUDA, "the persistent solver does not fit on this device");
    void* args[] = {(void*)&P};
    CU(cudaLaunchCooperativeKernel((const void*)cg_persistent_kernel<T, RECON, U1>, dim3(grid), dim3(PS_BLOCK), args, 0,
                                   c->stream));
    ++c->launches;
    return LQCD_OK;
}

template <typename T>
int launch_persistent(lqcd_ctx* c) {
    PrecBufs<T>& B = bufs<T>(c);
    PersistArgs<T> P{};
    P.D.g = c->g;
    P.D.W = B.W;
    P.D.Th = B.Th;
    set_policies<T>(c, P.D);
    P.st = c->st_dev;
    P.partials = c->partials;
    P.p = B.p;
    P.t = B.t;
    P.p_keep = B.p_keep;
    P.m = block_len(c);
    P.defer_base = defer_base(c);
    const bool r12 = B.recon_stored == 12;
    if (c->u1_on) return r12 ? launch_persistent_k<T, 12, 1>(c, P) : launch_persistent_k<T, 18, 1>(c, P);
    return r12 ? launch_persistent_k<T, 12, 0>(c, P) : launch_persistent_k<T, 18, 0>(c, P);
}

// The persistent solver pays when the iteration is bound by launch gaps and kernel tails rather than by bandwidth:
// lattices whose links AND solver vectors stay in L2.  Measured at 16^4, whole config-2 solve, us per iteration,
// persistent / launch path (four launches per iteration in a graph): two-row links (25 MB) 14.3 / 18.6, 18-real links
// (38 MB: with the residual ring and the x_i, p_i the working set no longer fits) 20.0 / 19.5.  Hence the bound on the
// stored links below.  Since the scalar steps ride in the sweeps on small lattices (dslash_kernel, FS = 1) the launch
// path takes 16.1 us with 18-real and 15.1 with two-row links there.  LQCD_OPT_PERSISTENT overrides.
#ifndef PERSIST_LINKS_MAX
#define PERSIST_LINKS_MAX (32u << 20)
#endif
template <typename T>
bool use_persistent(const lqcd_ctx* c) {
    if (c->slab || c->persistent_opt == 0) return false;
    if (!c->coop_launch || block_len(c) > PS_MAX_BLOCK) return false;
    // ... and enough sites to give most SMs a block of one site per thread (12^4: 41 blocks; 21 us per iteration against
    // 11.8 on the launch path)
    const bool fills = (long)((c->Vh + PS_BLOCK - 1) / PS_BLOCK) * 4 >= (long)c->num_sms * 3;
    return c->persistent_opt == 1 || (fills && links_bytes<T>(c, bufs_c<T>(c).recon_stored) <= PERSIST_LINKS_MAX);
}

bool over_p2p(const lqcd_ctx* c);

// the host looks at the stop flag every this many iterations: a whole number of blocks
int check_every(const lqcd_ctx* c) {
    long v = c->check_every ? (long)c->check_every : (long)(4000000 / (long)c->Vh);
    if (v < 1) v = 1;
    if (!c->check_every && v > 64) v = 64;
    // peer-memory transport with a time limit on the peers: the host runs two batches ahead of the device, and when a
    // peer is gone everything it has enqueued sits behind one stream wait.  Keep that well below the depth at which a
    // launch call itself blocks (there the time limit could not act): ~14 operations per iteration.
    if (!c->check_every && over_p2p(c) && c->comm_timeout > 0.0 && v > 16) v = 16;
    const long m = block_len(c);
    return (int)((v + m - 1) / m * m);
}

template <typename T>
int build_graph(lqcd_ctx* c, int iters, int rational) {
    (void)rational;                  // the kernels read the mode from the device state
    drop_graph<T>(c);
    PrecBufs<T>& B = bufs<T>(c);
    cudaGraph_t graph = nullptr;
    const long long before = c->launches;
    CU(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
    int rc_it = LQCD_OK;
    for (int i = 0; i < iters && !rc_it; ++i) rc_it = launch_cg_iteration<T>(c, i % block_len(c));
    cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    B.graph_launches = (int)(c->launches - before);
    c->launches = before;     // capturing is not launching
    if (rc_it) {
        if (graph) cudaGraphDestroy(graph);
        return rc_it;
    }
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "graph capture failed: %s", cudaGetErrorString(e));
    e = cudaGraphInstantiate(&B.graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) {
        B.graph_exec = nullptr;
        return fail(c, LQCD_ECUDA, "graph instantiate failed: %s", cudaGetErrorString(e));
    }
    B.graph_iters = iters;
    B.graph_rational = rational;
    B.graph_block = block_len(c);
    return LQCD_OK;
}

template <typename T>
int check_ctx_gauge(lqcd_ctx* c) {
    if (!bufs<T>(c).recon_stored)
        return fail(c, LQCD_ENOGAUGE, "no %s-precision gauge field stored (lqcd_set_gauge, LQCD_OPT_LINK_PRECISIONS)",
                    sizeof(T) == 8 ? "double" : "single");
    if (c->u1_on && !bufs<T>(c).u1_stored)
        return fail(c, LQCD_ENOGAUGE, "U(1) phases are on but not stored in %s precision (lqcd_set_u1_phases after "
                    "LQCD_OPT_LINK_PRECISIONS)", sizeof(T) == 8 ? "double" : "single");
    return LQCD_OK;
}

template <typename T>
int ensure_stage(lqcd_ctx* c, int nx) {
    int rc;
    PrecBufs<T>& B = bufs<T>(c);
    if (!B.stage_b && (rc = dev_alloc_own(c, (void**)&B.stage_b, vec_bytes<T>(c)))) return rc;
    while (B.n_stage_x < nx) {
        if ((rc = dev_alloc_own(c, (void**)&B.stage_x[B.n_stage_x], vec_bytes<T>(c)))) return rc;
        ++B.n_stage_x;
    }
    return LQCD_OK;
}

// Store the links in precision T (step A1).  `links` is the canonical double-precision field on the device.
template <typename T>
int store_gauge(lqcd_ctx* c, const double* links, int recon) {
    int rc;
    PrecBufs<T>& B = bufs<T>(c);
    const size_t need = links_bytes<T>(c, recon);
    if (!B.W || B.W_bytes < need) {
        if (B.W && !c->arena) dev_free_owned(c, B.W);
        B.W = nullptr;
        B.recon_stored = 0;
        const size_t want = c->arena ? links_bytes<T>(c, 18) : need;   // an arena slot is sized for either format
        if ((rc = dev_alloc(c, (void**)&B.W, want))) return rc;
        B.W_bytes = align_up(want);
    }
    B.recon_stored = 0;
    CU(cudaMemsetAsync(c->dev_max, 0, sizeof(double), c->stream));
    const size_t nthreads = 8 * c->Vh;
    const int grid = (int)((nthreads + 255) / 256);
    if (recon == 12)
        repack_gauge_kernel<T, 12><<<grid, 256, 0, c->stream>>>(c->g, (const double2*)links, B.W, c->dev_max);
    else
        repack_gauge_kernel<T, 18><<<grid, 256, 0, c->stream>>>(c->g, (const double2*)links, B.W, c->dev_max);
    ++c->launches;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(c->max_host, c->dev_max, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (recon == 12 && !(*c->max_host <= 1e-12))
        return fail(c, LQCD_ENOTSU3, "RECON=12 but max|r2 - conj(r0 x r1)| = %.3e > 1e-12", *c->max_host);
    if (c->slab) {
        // the backward t-hop of my lowest time slice needs the t-links that leave the slice below it: the top
        // t-links of rank-1, sent up the ring once (both origin parities, NE elements, stored format)
        const int NE = (recon == 12) ? 6 : 9;
        const size_t face = face_sites(c), vh = c->Vh;
        const size_t n = (size_t)2 * NE * face;
        if (!B.Wt_lo) {
            const size_t n18 = (size_t)2 * 9 * face;             // sized for either format
            if ((rc = dev_alloc(c, (void**)&B.Wt_lo, n18 * sizeof(V2<T>)))) return rc;
            if ((rc = dev_alloc(c, (void**)&B.Wt_send, 2 * n18 * sizeof(V2<T>)))) return rc;
        }
        const size_t row = face * sizeof(V2<T>);
        // rows (3*2 + parity)*NE + e of W, last time slice
        CU(cudaMemcpy2DAsync(B.Wt_send, row, B.W + (size_t)6 * NE * vh + (vh - face), vh * sizeof(V2<T>), row, 2 * NE,
                             cudaMemcpyDeviceToDevice, c->stream));
        CU(cudaEventRecord(c->ev_pack, c->stream));
        CU(cudaStreamWaitEvent(c->comm_stream, c->ev_pack, 0));
        V2<T>* dummy = B.Wt_send + (size_t)2 * 9 * face;        // what comes down the ring is not needed
        if ((rc = comm_exchange(c, B.Wt_send, B.Wt_send, B.Wt_lo, dummy, n * sizeof(V2<T>)))) return rc;
        CU(cudaStreamSynchronize(c->comm_stream));
        // first use of the all-reduce here, outside any stream capture: a transport that sets up connections or
        // buffers lazily (NCCL) has then done so before the CG iteration is captured into a CUDA graph
        CU(cudaMemsetAsync(c->red, 0, 2 * sizeof(double), c->stream));
        if ((rc = comm_allreduce(c))) return rc;
        CU(cudaStreamSynchronize(c->stream));
    }
    B.recon_stored = recon;
    return LQCD_OK;
}

// Store the U(1) angles in precision T: canonical theta[mu][lex] -> Th[(mu*2+par)*Vh + k].
template <typename T>
int store_theta(lqcd_ctx* c, const double* theta) {
    int rc;
    PrecBufs<T>& B = bufs<T>(c);
    B.u1_stored = 0;
    if (!B.Th && (rc = dev_alloc(c, (void**)&B.Th, (size_t)8 * c->Vh * sizeof(T)))) return rc;
    const size_t nthreads = 8 * c->Vh;
    repack_theta_kernel<T><<<(int)((nthreads + 255) / 256), 256, 0, c->stream>>>(c->g, theta, B.Th);
    ++c->launches;
    CU(cudaGetLastError());
    if (c->slab) {
        // the angles of the t-links that leave the slice below the slab (cf. the link halo in store_gauge)
        const size_t face = face_sites(c), vh = c->Vh;
        if (!B.Th_lo) {
            if ((rc = dev_alloc(c, (void**)&B.Th_lo, 2 * face * sizeof(T)))) return rc;
            if ((rc = dev_alloc(c, (void**)&B.Th_send, 4 * face * sizeof(T)))) return rc;
        }
        // rows (3*2 + parity) of Th, last time slice
        CU(cudaMemcpy2DAsync(B.Th_send, face * sizeof(T), B.Th + (size_t)6 * vh + (vh - face), vh * sizeof(T),
                             face * sizeof(T), 2, cudaMemcpyDeviceToDevice, c->stream));
        CU(cudaEventRecord(c->ev_pack, c->stream));
        CU(cudaStreamWaitEvent(c->comm_stream, c->ev_pack, 0));
        if ((rc = comm_exchange(c, B.Th_send, B.Th_send, B.Th_lo, B.Th_send + 2 * face, 2 * face * sizeof(T)))) return rc;
        CU(cudaStreamSynchronize(c->comm_stream));
    }
    B.u1_stored = 1;
    return LQCD_OK;
}

// release the stored links of precision T (no longer requested by LQCD_OPT_LINK_PRECISIONS)
template <typename T>
void release_gauge(lqcd_ctx* c) {
    PrecBufs<T>& B = bufs<T>(c);
    B.recon_stored = 0;
    if (B.W && !c->arena) {
        dev_free_owned(c, B.W);
        B.W = nullptr;
        B.W_bytes = 0;
    }
}

}  // namespace

extern "C" {

lqcd_ctx* lqcd_create(int Lx, int Ly, int Lz, int Lt) {
    const int L[4] = {Lx, Ly, Lz, Lt};
    for (int i = 0; i < 4; ++i)
        if (L[i] < 2 || (L[i] & 1)) {
            snprintf(g_create_error, sizeof(g_create_error), "extent %d = %d must be even and >= 2", i, L[i]);
            return nullptr;
        }
    const double vol = (double)Lx * Ly * Lz * Lt;
    if (vol / 2 >= 2147483648.0 / 4) {       // k, and k + stride, must stay below 2^31
        snprintf(g_create_error, sizeof(g_create_error), "volume too large for 32-bit site indices");
        return nullptr;
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        snprintf(g_create_error, sizeof(g_create_error), "no usable CUDA device: %s", cudaGetErrorString(e));
        return nullptr;
    }
    lqcd_ctx* c = new (std::nothrow) lqcd_ctx();
    if (!c) {
        snprintf(g_create_error, sizeof(g_create_error), "out of host memory");
        return nullptr;
    }
    for (int i = 0; i < 4; ++i) c->L[i] = L[i];
    c->V = (size_t)Lx * Ly * Lz * Lt;
    c->Vh = c->V / 2;
    Geom& g = c->g;
    g.Lxh = Lx / 2;
    g.Ly = Ly;
    g.Lz = Lz;
    g.Lt = Lt;
    g.Vh = (int)c->Vh;
    g.sy = g.Lxh;
    g.sz = g.Lxh * Ly;
    g.st = g.Lxh * Ly * Lz;
    g.dxh = make_fastdiv((uint32_t)g.Lxh);
    g.dy = make_fastdiv((uint32_t)Ly);
    g.dz = make_fastdiv((uint32_t)Lz);
    g.antiperiodic = 1;
    g.t_off = 0;
    g.Lt_glob = Lt;
    c->slab = 0;
    c->rank = 0;
    c->nranks = 1;
    c->has_comm = false;
    c->device = dev;
    c->num_sms = prop.multiProcessorCount;
    c->coop_launch = prop.cooperativeLaunch;
    c->stream = nullptr;
    c->mass = 0.0;
    c->recon_opt = 18;
    c->prec_opt = LQCD_PREC_F64;
    c->u1_on = 0;
    c->max_iter = 100000;
    c->check_every = 0;
    c->use_graph = 1;
    c->shift_block_opt = 0;
    c->persistent_opt = -1;
    c->comm_timeout = 120.0;
    c->err[0] = 0;
    return c;
}

void lqcd_destroy(lqcd_ctx* c) {
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    drop_graphs(c);
    for (void* p : c->owned) cudaFree(p);
    if (c->st_host) cudaFreeHost(c->st_host);
    if (c->flag_host) cudaFreeHost(c->flag_host);
    if (c->max_host) cudaFreeHost(c->max_host);
    if (c->nccl.comm) {
        lqcd_nccl::Api* a = lqcd_nccl::api(nullptr);
        if (a) a->CommDestroy(c->nccl.comm);
    }
    lqcd_p2p::destroy(&c->p2p);
    if (c->host_stage) cudaFreeHost(c->host_stage);
    if (c->red_host) cudaFreeHost(c->red_host);
    if (c->comm_stream) cudaStreamDestroy(c->comm_stream);
    cudaEvent_t evs[] = {c->ev_pack, c->ev_halo, c->ev[0], c->ev[1], c->ev_t0, c->ev_t1, c->ev_m0, c->ev_m1};
    for (cudaEvent_t e : evs)
        if (e) cudaEventDestroy(e);
    cudaGetLastError();
    delete c;
}

const char* lqcd_last_error(const lqcd_ctx* c) { return c ? c->err : g_create_error; }

lqcd_ctx* lqcd_create_slab(int Lx, int Ly, int Lz, int Lt_global, int rank, int nranks) {
    if (nranks < 1 || rank < 0 || rank >= nranks) {
        snprintf(g_create_error, sizeof(g_create_error), "rank %d of %d is not a valid slab", rank, nranks);
        return nullptr;
    }
    if (Lt_global < 2 || Lt_global % nranks != 0 || ((Lt_global / nranks) & 1)) {
        snprintf(g_create_error, sizeof(g_create_error), "Lt = %d over %d ranks: every slab needs an even number of time slices",
                 Lt_global, nranks);
        return nullptr;
    }
    const int Lt_loc = Lt_global / nranks;
    lqcd_ctx* c = lqcd_create(Lx, Ly, Lz, Lt_loc);
    if (!c) return nullptr;
    c->slab = 1;
    c->rank = rank;
    c->nranks = nranks;
    c->g.t_off = rank * Lt_loc;
    c->g.Lt_glob = Lt_global;
    return c;
}

int lqcd_slab_info(const lqcd_ctx* c, int* rank, int* nranks, int* t_offset, int* Lt_global) {
    if (!c) return LQCD_EINVAL;
    if (rank) *rank = c->rank;
    if (nranks) *nranks = c->nranks;
    if (t_offset) *t_offset = c->g.t_off;
    if (Lt_global) *Lt_global = c->g.Lt_glob;
    return LQCD_OK;
}

int lqcd_set_comm(lqcd_ctx* c, const lqcd_comm_ops* ops) {
    if (!c) return LQCD_EINVAL;
    if (!c->slab) return fail(c, LQCD_EINVAL, "not a slab context (lqcd_create_slab)");
    if (!ops || !ops->exchange || !ops->allreduce_sum) return fail(c, LQCD_EINVAL, "transport functions missing");
    drop_graphs(c);
    c->comm = *ops;
    c->has_comm = true;
    return LQCD_OK;
}

int lqcd_nccl_unique_id(void* id) {
    if (!id) return LQCD_EINVAL;
    const char* why = nullptr;
    lqcd_nccl::Api* a = lqcd_nccl::api(&why);
    if (!a) {
        snprintf(g_create_error, sizeof(g_create_error), "NCCL unavailable: %s", why ? why : "?");
        return LQCD_ECOMM;
    }
    lqcd_nccl::unique_id u;
    const int rc = a->GetUniqueId(&u);
    if (rc) {
        snprintf(g_create_error, sizeof(g_create_error), "ncclGetUniqueId: %s", a->GetErrorString(rc));
        return LQCD_ECOMM;
    }
    memcpy(id, &u, sizeof(u));
    return LQCD_OK;
}

int lqcd_comm_init_nccl(lqcd_ctx* c, const void* id) {
    if (!c) return LQCD_EINVAL;
    if (!c->slab) return fail(c, LQCD_EINVAL, "not a slab context (lqcd_create_slab)");
    if (!id) return fail(c, LQCD_EINVAL, "id is NULL");
    if (c->nccl.comm) return fail(c, LQCD_EINVAL, "NCCL transport already initialised");
    const char* why = nullptr;
    lqcd_nccl::Api* a = lqcd_nccl::api(&why);
    if (!a) return fail(c, LQCD_ECOMM, "NCCL unavailable: %s", why ? why : "?");
    lqcd_nccl::unique_id u;
    memcpy(&u, id, sizeof(u));
    c->nccl.rank = c->rank;
    c->nccl.nranks = c->nranks;
    const int rc = a->CommInitRank(&c->nccl.comm, c->nranks, u, c->rank);
    if (rc) {
        c->nccl.comm = nullptr;
        return fail(c, LQCD_ECOMM, "ncclCommInitRank: %s", a->GetErrorString(rc));
    }
    lqcd_comm_ops ops;
    ops.user = &c->nccl;
    ops.exchange = lqcd_nccl::exchange;
    ops.allreduce_sum = lqcd_nccl::allreduce_sum;
    ops.host_staged = 0;
    ops.graph_safe = 1;
    return lqcd_set_comm(c, &ops);
}

int lqcd_p2p_export(lqcd_ctx* c, void* handle) {
    if (!c) return LQCD_EINVAL;
    if (!c->slab) return fail(c, LQCD_EINVAL, "not a slab context (lqcd_create_slab)");
    if (!handle) return fail(c, LQCD_EINVAL, "handle is NULL");
    // a face buffer holds the largest message of the path: the t-links of one face, both parities, 18 reals, double
    const size_t cap = (size_t)2 * 9 * face_sites(c) * sizeof(double2);
    lqcd_p2p::Blob b;
    if (lqcd_p2p::create_window(&c->p2p, c->rank, c->nranks, cap, &b)) return fail(c, LQCD_ECOMM, "peer-memory transport: %s", c->p2p.error);
    memcpy(handle, &b, sizeof(b));
    return LQCD_OK;
}

int lqcd_comm_init_p2p(lqcd_ctx* c, const void* handles) {
    if (!c) return LQCD_EINVAL;
    if (!c->slab) return fail(c, LQCD_EINVAL, "not a slab context (lqcd_create_slab)");
    if (!handles) return fail(c, LQCD_EINVAL, "handles is NULL");
    if (c->p2p.active) return fail(c, LQCD_EINVAL, "peer-memory transport already initialised");
    static_assert(sizeof(lqcd_p2p::Blob) == LQCD_P2P_HANDLE_BYTES, "LQCD_P2P_HANDLE_BYTES");
    std::vector<lqcd_p2p::Blob> blobs((size_t)c->nranks);
    memcpy(blobs.data(), handles, blobs.size() * sizeof(lqcd_p2p::Blob));
    if (lqcd_p2p::connect(&c->p2p, blobs.data())) return fail(c, LQCD_ECOMM, "peer-memory transport: %s", c->p2p.error);
    lqcd_comm_ops ops;
    ops.user = &c->p2p;
    ops.exchange = lqcd_p2p::exchange;
    ops.allreduce_sum = lqcd_p2p::allreduce_sum;
    ops.host_staged = 0;
    // The stream memory operations can be captured (values are constants, addresses depend on the generation only), and
    // a captured iteration was run and was correct -- and slower than plain launches at every size tried (one rank, us
    // per iteration, graph / plain: 16^4 72.0 / 71.9, 32^4 271 / 254, 48^4 1191 / 1170): launched plainly.
    ops.graph_safe = 0;
    return lqcd_set_comm(c, &ops);
}

int lqcd_set_stream(lqcd_ctx* c, void* cuda_stream) {
    if (!c) return LQCD_EINVAL;
    c->stream = (cudaStream_t)cuda_stream;
    return LQCD_OK;
}

int lqcd_set_option(lqcd_ctx* c, int key, double v) {
    if (!c) return LQCD_EINVAL;
    switch (key) {
        case LQCD_OPT_MASS:
            if (!std::isfinite(v)) return fail(c, LQCD_EINVAL, "mass must be finite");
            c->mass = v;
            break;
        case LQCD_OPT_ANTIPERIODIC_T:
            if (v != 0.0 && v != 1.0) return fail(c, LQCD_EINVAL, "ANTIPERIODIC_T must be 0 or 1");
            c->g.antiperiodic = (int)v;
            drop_graphs(c);       // Geom is a kernel argument baked into the graph
            break;
        case LQCD_OPT_RECON:
            if (v != 18.0 && v != 12.0) return fail(c, LQCD_EINVAL, "RECON must be 18 or 12");
            c->recon_opt = (int)v;
            break;
        case LQCD_OPT_MAX_ITER:
            if (!(v >= 1.0) || v > 2.0e9) return fail(c, LQCD_EINVAL, "MAX_ITER must be in [1, 2e9]");
            c->max_iter = (int)v;
            break;
        case LQCD_OPT_CHECK_EVERY:
            if (!(v >= 0.0) || v > 1.0e6) return fail(c, LQCD_EINVAL, "CHECK_EVERY must be in [0, 1e6]");
            c->check_every = (int)v;
            break;
        case LQCD_OPT_USE_GRAPH:
            if (v != 0.0 && v != 1.0) return fail(c, LQCD_EINVAL, "USE_GRAPH must be 0 or 1");
            c->use_graph = (int)v;
            break;
        case LQCD_OPT_SHIFT_BLOCK:
            if (!(v >= 0.0) || v > (double)LQCD_MAX_BLOCK || v != std::floor(v))
                return fail(c, LQCD_EINVAL, "SHIFT_BLOCK must be an integer in [1, %d], or 0 (chosen by the library)", LQCD_MAX_BLOCK);
            c->shift_block_opt = (int)v;
            break;
        case LQCD_OPT_PERSISTENT:
            if (v != -1.0 && v != 0.0 && v != 1.0) return fail(c, LQCD_EINVAL, "PERSISTENT must be -1 (auto), 0 or 1");
            c->persistent_opt = (int)v;
            break;
        case LQCD_OPT_COMM_TIMEOUT:
            if (!(v >= 0.0)) return fail(c, LQCD_EINVAL, "COMM_TIMEOUT must be >= 0 seconds (0: wait for ever)");
            c->comm_timeout = v;
            break;
        case LQCD_OPT_LINK_PRECISIONS:
            if (v != 1.0 && v != 2.0 && v != 3.0)
                return fail(c, LQCD_EINVAL, "LINK_PRECISIONS must be LQCD_PREC_F64 (1), LQCD_PREC_F32 (2) or both (3)");
            c->prec_opt = (int)v;
            break;
        default:
            return fail(c, LQCD_EINVAL, "unknown option key %d", key);
    }
    return LQCD_OK;
}

int lqcd_get_option(const lqcd_ctx* c, int key, double* v) {
    if (!c || !v) return LQCD_EINVAL;
    switch (key) {
        case LQCD_OPT_MASS: *v = c->mass; break;
        case LQCD_OPT_ANTIPERIODIC_T: *v = c->g.antiperiodic; break;
        case LQCD_OPT_RECON: *v = c->recon_opt; break;
        case LQCD_OPT_MAX_ITER: *v = c->max_iter; break;
        case LQCD_OPT_CHECK_EVERY: *v = check_every(c); break;
        case LQCD_OPT_SHIFT_BLOCK: *v = block_len(c); break;
        case LQCD_OPT_USE_GRAPH: *v = c->use_graph; break;
        case LQCD_OPT_LINK_PRECISIONS: *v = c->prec_opt; break;
        case LQCD_OPT_PERSISTENT: *v = c->persistent_opt; break;
        case LQCD_OPT_COMM_TIMEOUT: *v = c->comm_timeout; break;
        default: return LQCD_EINVAL;
    }
    return LQCD_OK;
}

size_t lqcd_workspace_bytes(const lqcd_ctx* c, int nshift) {
    if (!c || nshift < 1 || nshift > LQCD_MAX_SHIFTS) return 0;
    size_t b = 0;
    if (c->prec_opt & LQCD_PREC_F64)
        b += align_up(links_bytes<double>(c, 18)) + align_up(vec_bytes<double>(c)) * (size_t)(3 + block_len(c) + (nshift - 1));
    if (c->prec_opt & LQCD_PREC_F32)
        b += align_up(links_bytes<float>(c, 18)) + align_up(vec_bytes<float>(c)) * (size_t)(3 + block_len(c) + (nshift - 1));
    if (c->prec_opt & LQCD_PREC_F64) b += align_up((size_t)8 * c->Vh * sizeof(double));   // U(1) angles, if set
    if (c->prec_opt & LQCD_PREC_F32) b += align_up((size_t)8 * c->Vh * sizeof(float));
    b += align_up(sizeof(CgState)) + align_up(sizeof(double)) + align_up(2 * sizeof(double));
    if (c->slab) {
        const size_t face = face_sites(c);
        if (c->prec_opt & LQCD_PREC_F64) b += 2 * align_up(6 * face * sizeof(double2)) + align_up(18 * face * sizeof(double2)) + align_up(36 * face * sizeof(double2));
        if (c->prec_opt & LQCD_PREC_F32) b += 2 * align_up(6 * face * sizeof(float2)) + align_up(18 * face * sizeof(float2)) + align_up(36 * face * sizeof(float2));
    }
    b += align_up(n_partials_needed(c) * sizeof(double));
    return b;
}

int lqcd_set_workspace(lqcd_ctx* c, void* dev, size_t bytes) {
    if (!c) return LQCD_EINVAL;
    if (c->d.recon_stored || c->f.recon_stored || c->basics || !c->owned.empty())
        return fail(c, LQCD_EINVAL, "lqcd_set_workspace must be called before any other device work on the context");
    if (!dev || ((uintptr_t)dev % ALIGN) != 0) return fail(c, LQCD_EINVAL, "workspace must be a 256-byte aligned device pointer");
    c->arena = (char*)dev;
    c->arena_bytes = bytes;
    c->arena_used = 0;
    return LQCD_OK;
}

int lqcd_set_gauge(lqcd_ctx* c, const double* links) {
    if (!c) return LQCD_EINVAL;
    if (!links) return fail(c, LQCD_EINVAL, "links is NULL");
    if (c->slab && !c->has_comm)
        return fail(c, LQCD_ECOMM, "slab context: set a transport (lqcd_comm_init_nccl / lqcd_set_comm) before lqcd_set_gauge");
    int rc;
    if ((rc = ensure_basics(c))) return rc;
    drop_graphs(c);
    c->d.recon_stored = 0;
    c->f.recon_stored = 0;
    if (c->prec_opt & LQCD_PREC_F64) {
        if ((rc = store_gauge<double>(c, links, c->recon_opt))) return rc;
    } else {
        release_gauge<double>(c);
    }
    if (c->prec_opt & LQCD_PREC_F32) {
        if ((rc = store_gauge<float>(c, links, c->recon_opt))) {
            c->d.recon_stored = 0;
            return rc;
        }
    } else {
        release_gauge<float>(c);
    }
    return LQCD_OK;
}

int lqcd_set_u1_phases(lqcd_ctx* c, const double* theta) {
    if (!c) return LQCD_EINVAL;
    if (c->slab && theta && !c->has_comm)
        return fail(c, LQCD_ECOMM, "slab context: set a transport before lqcd_set_u1_phases");
    int rc;
    if ((rc = ensure_basics(c))) return rc;
    drop_graphs(c);           // the kernel variant and its arguments are baked into the graph
    c->u1_on = 0;
    c->d.u1_stored = c->f.u1_stored = 0;
    if (!theta) return LQCD_OK;
    if ((c->prec_opt & LQCD_PREC_F64) && (rc = store_theta<double>(c, theta))) return rc;
    if ((c->prec_opt & LQCD_PREC_F32) && (rc = store_theta<float>(c, theta))) return rc;
    CU(cudaStreamSynchronize(c->stream));       // theta may be freed by the caller on return
    c->u1_on = 1;
    return LQCD_OK;
}

int lqcd_set_u1_phases_host(lqcd_ctx* c, const double* theta) {
    if (!c) return LQCD_EINVAL;
    if (!theta) return lqcd_set_u1_phases(c, nullptr);
    const size_t bytes = (size_t)4 * c->V * sizeof(double);
    void* tmp = nullptr;
    cudaError_t e = cudaMalloc(&tmp, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(c, LQCD_ENOMEM, "cudaMalloc(%zu) for the canonical U(1) angles failed", bytes);
    }
    e = cudaMemcpyAsync(tmp, theta, bytes, cudaMemcpyHostToDevice, c->stream);
    int rc = LQCD_OK;
    if (e != cudaSuccess) rc = fail(c, LQCD_ECUDA, "copy of the U(1) angles failed: %s", cudaGetErrorString(e));
    if (!rc) rc = lqcd_set_u1_phases(c, (const double*)tmp);
    cudaStreamSynchronize(c->stream);
    cudaFree(tmp);
    return rc;
}

int lqcd_set_gauge_host(lqcd_ctx* c, const double* links) {
    if (!c) return LQCD_EINVAL;
    if (!links) return fail(c, LQCD_EINVAL, "links is NULL");
    const size_t bytes = (size_t)4 * c->V * 9 * sizeof(double2);
    void* tmp = nullptr;
    cudaError_t e = cudaMalloc(&tmp, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(c, LQCD_ENOMEM, "cudaMalloc(%zu) for the canonical links failed", bytes);
    }
    e = cudaMemcpyAsync(tmp, links, bytes, cudaMemcpyHostToDevice, c->stream);
    int rc = LQCD_OK;
    if (e != cudaSuccess) rc = fail(c, LQCD_ECUDA, "copy of the links failed: %s", cudaGetErrorString(e));
    if (!rc) rc = lqcd_set_gauge(c, (const double*)tmp);
    cudaStreamSynchronize(c->stream);
    cudaFree(tmp);
    return rc;
}

}  // extern "C"

namespace {

template <typename T>
int apply_d(lqcd_ctx* c, T* out, const T* in, int par) {
    if (!c) return LQCD_EINVAL;
    if (!out || !in) return fail(c, LQCD_EINVAL, "NULL vector");
    if (out == in) return fail(c, LQCD_EINVAL, "in and out must not alias");
    int rc;
    if ((rc = check_ctx_gauge<T>(c))) return rc;
    if (c->slab) {
        if ((rc = ensure_basics(c))) return rc;
        return slab_dslash<T>(c, 0, (V2<T>*)out, (const V2<T>*)in, par, nullptr, 0.0);
    }
    launch_dslash<T>(c, 0, (V2<T>*)out, (const V2<T>*)in, par, nullptr, 0.0, 0);
    CU(cudaGetLastError());
    return LQCD_OK;
}

template <typename T>
int apply_d_host(lqcd_ctx* c, T* out, const T* in, int par) {
    if (!c) return LQCD_EINVAL;
    if (!out || !in) return fail(c, LQCD_EINVAL, "NULL vector");
    int rc;
    if ((rc = check_ctx_gauge<T>(c))) return rc;
    if ((rc = ensure_stage<T>(c, 1))) return rc;
    PrecBufs<T>& B = bufs<T>(c);
    CU(cudaMemcpyAsync(B.stage_b, in, vec_bytes<T>(c), cudaMemcpyHostToDevice, c->stream));
    if ((rc = apply_d<T>(c, (T*)B.stage_x[0], (const T*)B.stage_b, par))) return rc;
    CU(cudaMemcpyAsync(out, B.stage_x[0], vec_bytes<T>(c), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return LQCD_OK;
}

template <typename T>
int apply_mdagm(lqcd_ctx* c, T* out_even, const T* in_even, double sigma) {
    if (!c) return LQCD_EINVAL;
    if (!out_even || !in_even) return fail(c, LQCD_EINVAL, "NULL vector");
    if (out_even == in_even) return fail(c, LQCD_EINVAL, "in and out must not alias");
    int rc;
    if ((rc = check_ctx_gauge<T>(c))) return rc;
    if ((rc = ensure_tmp<T>(c))) return rc;
    PrecBufs<T>& B = bufs<T>(c);
    if (c->slab) {
        if ((rc = slab_dslash<T>(c, 0, B.t, (const V2<T>*)in_even, 1, nullptr, 0.0))) return rc;
        return slab_dslash<T>(c, 2, (V2<T>*)out_even, B.t, 0, (const V2<T>*)in_even, c->mass * c->mass + sigma);
    }
    launch_dslash<T>(c, 0, B.t, (const V2<T>*)in_even, 1, nullptr, 0.0, 0);
    launch_dslash<T>(c, 2, (V2<T>*)out_even, B.t, 0, (const V2<T>*)in_even, c->mass * c->mass + sigma, 0);
    CU(cudaGetLastError());
    return LQCD_OK;
}

// The solver behind lqcd_mshift_cg (x != NULL: every x[i] is stored) and lqcd_rational_apply (y != NULL:
// only y = alpha0 b + sum_i alpha[i] x_i is accumulated), in precision T.
// ---- a solve over the peer-memory transport must not wait for ever --------------------------------------------------
// Over that transport a rank waits for its peers with stream memory operations on its own window (p2p.cuh).  A peer
// that has failed releases the others by marking their words (lqcd_p2p::poison) -- but a peer whose process was killed
// marks nothing.  So on such a context the host does not block in cudaEventSynchronize: it polls, and after
// LQCD_OPT_COMM_TIMEOUT seconds without the awaited batch completing it gives up: it releases its own streams and its
// peers and the solve returns LQCD_ECOMM.
bool over_p2p(const lqcd_ctx* c) { return c->slab && c->p2p.active && c->comm.user == (const void*)&c->p2p; }

int wait_event_watched(lqcd_ctx* c, cudaEvent_t ev, bool* timed_out) {
    *timed_out = false;
    if (!over_p2p(c) || !(c->comm_timeout > 0.0)) {
        CU(cudaEventSynchronize(ev));
        return LQCD_OK;
    }
    const auto t0 = std::chrono::steady_clock::now();
    for (;;) {
        const cudaError_t e = cudaEventQuery(ev);
        if (e == cudaSuccess) return LQCD_OK;
        if (e != cudaErrorNotReady) CU(e);
        const double waited = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
        if (waited > c->comm_timeout) {
            *timed_out = true;
            return LQCD_OK;
        }
        if (waited > 2e-4) std::this_thread::sleep_for(std::chrono::microseconds(50));     // spin first: batches are short
    }
}

// the awaited work did not complete in time: release everybody (this rank included), let this rank's streams drain
int give_up_waiting(lqcd_ctx* c) {
    lqcd_p2p::poison(&c->p2p, true);
    bool again = false;
    cudaEvent_t ev = c->ev[0];
    if (cudaEventRecord(ev, c->stream) == cudaSuccess) wait_event_watched(c, ev, &again);
    cudaGetLastError();
    return fail(c, LQCD_ECOMM, "peer-memory transport: no sign of a peer rank for %.1f s (LQCD_OPT_COMM_TIMEOUT)%s; the "
                "context can only be destroyed", c->comm_timeout, again ? ", and this rank's stream did not drain" : "");
}

template <typename T>
int solve_impl(lqcd_ctx* c, const T* b_even, const double* shifts, int nshift, double tol, T* const* x, T* y, double alpha0,
               const double* alpha);

template <typename T>
int solve(lqcd_ctx* c, const T* b_even, const double* shifts, int nshift, double tol, T* const* x, T* y, double alpha0,
          const double* alpha) {
    if (c && c->p2p.dead)
        return fail(c, LQCD_ECOMM, "the peer-memory transport of this context has failed (%s): destroy the context on every "
                    "rank and set the ranks up again", c->p2p.error);
    const int rc = solve_impl<T>(c, b_even, shifts, nshift, tol, x, y, alpha0, alpha);
    // a rank that leaves a solve early takes its peers with it instead of leaving them waiting for its faces and sums
    if (c && over_p2p(c) && (rc == LQCD_ECOMM || rc == LQCD_ECUDA)) lqcd_p2p::poison(&c->p2p, false);
    return rc;
}

template <typename T>
int solve_impl(lqcd_ctx* c, const T* b_even, const double* shifts, int nshift, double tol, T* const* x, T* y, double alpha0,
               const double* alpha) {
    if (!c) return LQCD_EINVAL;
    if (!b_even || !shifts || (!x && !y) || (y && !alpha)) return fail(c, LQCD_EINVAL, "NULL argument");
    if (nshift < 1 || nshift > LQCD_MAX_SHIFTS) return fail(c, LQCD_EINVAL, "nshift must be in [1, %d]", LQCD_MAX_SHIFTS);
    if (!(tol > 0.0) || !std::isfinite(tol)) return fail(c, LQCD_EINVAL, "tol must be positive");
    for (int i = 0; i < nshift; ++i) {
        if (!(shifts[i] >= 0.0) || !std::isfinite(shifts[i])) return fail(c, LQCD_EINVAL, "shift %d must be >= 0", i);
        if (y) {
            if (!std::isfinite(alpha[i])) return fail(c, LQCD_EINVAL, "alpha[%d] must be finite", i);
            continue;
        }
        if (!x[i] || (const T*)x[i] == b_even) return fail(c, LQCD_EINVAL, "x[%d] is NULL or aliases b", i);
        for (int j = 0; j < i; ++j)
            if (x[j] == x[i]) return fail(c, LQCD_EINVAL, "x[%d] aliases x[%d]", i, j);
    }
    if (y && (y == b_even || !std::isfinite(alpha0))) return fail(c, LQCD_EINVAL, "y aliases b, or alpha0 is not finite");
    const int rational = y ? 1 : 0;
    int rc;
    if ((rc = check_ctx_gauge<T>(c))) return rc;
    if ((rc = ensure_solver<T>(c, nshift))) return rc;
    if (c->slab && (rc = ensure_halo<T>(c))) return rc;      // nothing may be allocated while the graph is captured
    PrecBufs<T>& B = bufs<T>(c);

    // base system = smallest shift (R5); ties: the first
    int i0 = 0;
    for (int i = 1; i < nshift; ++i)
        if (shifts[i] < shifts[i0]) i0 = i;

    CgState* h = c->st_host;
    memset(h, 0, sizeof(CgState));
    h->nshift = nshift;
    h->i0 = i0;
    h->max_iter = c->max_iter;
    h->c0 = c->mass * c->mass + shifts[i0];
    int extra = 0;
    for (int i = 0; i < nshift; ++i) {
        h->delta[i] = shifts[i] - shifts[i0];
        h->x[i] = rational ? nullptr : (void*)x[i];
        h->alpha[i] = rational ? alpha[i] : 0.0;
        h->p[i] = (i == i0) ? (void*)B.p : (void*)B.pextra[extra++];
    }
    const int m = block_len(c);
    h->blk_m = m;
    for (int l = 0; l < m; ++l) h->hist[l] = (void*)B.hist[l];
    h->rational = rational;
    h->alpha0 = alpha0;
    h->y = (void*)y;
    h->defer_base = defer_base(c);
    h->p_keep = (void*)B.p_keep;
    h->b_src = (const void*)b_even;
    const size_t n = c->Vh * 3;
    CU(cudaMemcpyAsync(c->st_dev, h, sizeof(CgState), cudaMemcpyHostToDevice, c->stream));
    CU(cudaEventRecord(c->ev_t0, c->stream));
    if (c->slab) {
        if (!c->has_comm) return fail(c, LQCD_ECOMM, "slab context without a transport (lqcd_comm_init_nccl / lqcd_set_comm)");
        cg_init_kernel<T, false><<<cg_grid(c), CG_BLOCK, 0, c->stream>>>((const V2<T>*)b_even, B.hist[m - 1], c->st_dev,
                                                                         c->partials, n, tol);
        ++c->launches;
        if ((rc = slab_reduce_step(c, cg_grid(c), 0, tol, 0))) return rc;
    } else {
        cg_init_kernel<T><<<cg_grid(c), CG_BLOCK, 0, c->stream>>>((const V2<T>*)b_even, B.hist[m - 1], c->st_dev, c->partials, n, tol);
        ++c->launches;
    }
    CU(cudaGetLastError());

    const int ce = check_every(c);
    bool persistent = use_persistent<T>(c);
    if (c->persistent_opt == 1 && !persistent)
        return fail(c, LQCD_EINVAL, "LQCD_OPT_PERSISTENT = 1, but the persistent kernel cannot run this solve (%s)",
                    c->slab ? "slab context" : !c->coop_launch ? "no cooperative launches on this device"
                                                               : "LQCD_OPT_SHIFT_BLOCK above 16");
    c->flag_host[0] = c->flag_host[1] = 0;
    c->last_replays = 0;
    bool done = false;
    if (persistent) {
        // one cooperative kernel runs the iterations until the device-side stop (persist.cuh)
        rc = launch_persistent<T>(c);
        if (rc == LQCD_OK) {
            done = true;
        } else if (c->persistent_opt == 1) {
            return rc;
        } else {
            // the library chose this driver and the launch was refused (fewer blocks can be resident than the occupancy
            // query said: another context or MPS client on the device): nothing has run, take the other driver
            cudaGetLastError();
            persistent = false;
        }
    }
    // the legacy default stream cannot be captured: plain launches there
    // Slabs: a replayed graph does not keep the priority of the communication stream, so the border launches queue
    // behind the interior again; measured on one rank over NCCL, graph against plain launches, us per iteration:
    // 16^4 48.9 / 61.6, 32^4 256 / 246, 48^4 1175 / 1167 -- the graph pays only where launches are what limits
    const bool use_graph = !persistent && c->use_graph && c->stream != nullptr && c->stream != cudaStreamLegacy &&
                           (!c->slab || (c->comm.graph_safe && c->Vh <= SLAB_GRAPH_MAX_VH));
    if (use_graph && (B.graph_iters != ce || B.graph_block != m)) {
        if ((rc = build_graph<T>(c, ce, rational))) return rc;
    }
    c->last_path = persistent ? 2 : use_graph ? 1 : 0;
    // MAX_ITER is reached inside batch number ceil(MAX_ITER / ce) at the latest: nothing is launched beyond it (the
    // kernels of a launch whose solve is over return at once, but 2 x 20,000 empty blocks per iteration are not free)
    const long max_batches = ((long)c->max_iter + ce - 1) / ce;
    for (long batch = 0; batch < max_batches && !done; ++batch) {
        // the batch in which MAX_ITER falls is launched plainly, only as far as the cap: the iterations of a graph
        // replay beyond it would all return at once, at 27 us each (48^4)
        const long left = (long)c->max_iter - batch * ce;
        const int nit = (left < ce) ? (int)left : ce;       // the same on every rank of a slab decomposition
        if (use_graph && nit == ce) {
            CU(cudaGraphLaunch(B.graph_exec, c->stream));
            c->launches += B.graph_launches;
            ++c->last_replays;
        } else {
            for (int i = 0; i < nit; ++i)
                if ((rc = launch_cg_iteration<T>(c, i % m))) return rc;
            if (nit % m != 0) {                              // the stop falls inside a block: close it
                if (fused_scalar(c)) launch_reduce_scalar(c, 2, partials_k2(c));
                launch_flush<T>(c);
            }
            CU(cudaGetLastError());
        }
        const int slot = (int)(batch & 1);
        CU(cudaMemcpyAsync(&c->flag_host[slot], &c->st_dev->stop, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaEventRecord(c->ev[slot], c->stream));
        if (batch >= 1) {
            bool late = false;
            if ((rc = wait_event_watched(c, c->ev[slot ^ 1], &late))) return rc;
            if (late) return give_up_waiting(c);
            if (c->flag_host[slot ^ 1]) done = true;
        }
    }
    CU(cudaEventRecord(c->ev_t1, c->stream));
    CU(cudaMemcpyAsync(h, c->st_dev, sizeof(CgState), cudaMemcpyDeviceToHost, c->stream));
    {
        bool late = false;
        CU(cudaEventRecord(c->ev[0], c->stream));
        if ((rc = wait_event_watched(c, c->ev[0], &late))) return rc;
        if (late) return give_up_waiting(c);
    }
    CU(cudaStreamSynchronize(c->stream));
    CU(cudaEventElapsedTime(&c->last_ms, c->ev_t0, c->ev_t1));

    if (h->iter == 0 && !rational) {
        // nothing was ever accumulated (zero source, or breakdown in the first iteration): no sweep has written the x_i
        for (int i = 0; i < nshift; ++i) CU(cudaMemsetAsync(x[i], 0, n * sizeof(V2<T>), c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    c->last_iters = h->iter;
    c->last_i0 = i0;
    c->last_nshift = nshift;
    c->last_rel = (h->bb > 0.0) ? std::sqrt(h->rr / h->bb) : 0.0;
    for (int i = 0; i < nshift; ++i) c->last_freeze[i] = h->active[i] ? h->iter : h->freeze_iter[i];
    if (h->status == LQCD_ECOMM)
        return fail(c, LQCD_ECOMM, "peer-memory transport: a peer rank gave up during the solve (iteration %d); the context "
                    "can only be destroyed", h->iter);
    if (!h->stop) return fail(c, LQCD_ECUDA, "solver loop ended without the device raising its stop flag");
    if (h->status == LQCD_EBREAKDOWN) return fail(c, LQCD_EBREAKDOWN, "<p,Ap> = %g at iteration %d", h->pAp, h->iter);
    if (h->status == LQCD_ENOCONV)
        return fail(c, LQCD_ENOCONV, "no convergence in %d iterations, |r|/|b| = %.3e", h->iter, c->last_rel);
    return LQCD_OK;
}

template <typename T>
int solve_host(lqcd_ctx* c, const T* b_even, const double* shifts, int nshift, double tol, T* const* x, T* y,
               double alpha0, const double* alpha) {
    if (!c) return LQCD_EINVAL;
    if (!b_even || !shifts || (!x && !y)) return fail(c, LQCD_EINVAL, "NULL argument");
    if (nshift < 1 || nshift > LQCD_MAX_SHIFTS) return fail(c, LQCD_EINVAL, "nshift must be in [1, %d]", LQCD_MAX_SHIFTS);
    const int nout = y ? 1 : nshift;
    for (int i = 0; x && i < nshift; ++i)
        if (!x[i]) return fail(c, LQCD_EINVAL, "x[%d] is NULL", i);
    int rc;
    if ((rc = check_ctx_gauge<T>(c))) return rc;
    if ((rc = ensure_stage<T>(c, nout))) return rc;
    PrecBufs<T>& B = bufs<T>(c);
    CU(cudaMemcpyAsync(B.stage_b, b_even, vec_bytes<T>(c), cudaMemcpyHostToDevice, c->stream));
    T* xd[LQCD_MAX_SHIFTS];
    for (int i = 0; i < nout; ++i) xd[i] = (T*)B.stage_x[i];
    const int status = y ? solve<T>(c, (const T*)B.stage_b, shifts, nshift, tol, nullptr, xd[0], alpha0, alpha)
                         : solve<T>(c, (const T*)B.stage_b, shifts, nshift, tol, xd, nullptr, 0.0, nullptr);
    if (status != LQCD_OK && status != LQCD_ENOCONV) return status;
    for (int i = 0; i < nout; ++i)
        CU(cudaMemcpyAsync(y ? y : x[i], B.stage_x[i], vec_bytes<T>(c), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return status;
}

// ---- mixed precision (NEXT-2): float CG with double-precision reliable updates ---------------------------------
// One system (A + sigma) x = b, A = m^2 - D_eo D_oe, to the tolerance tol on the TRUE residual computed in double.
// x holds the initial guess on entry when have_guess (it is then improved), else it is overwritten.
// The float iterations run as the ordinary single-shift solver (same kernels, same CUDA graph); between batches of
// CHECK_EVERY iterations the host looks at the recurrence residual and triggers a reliable update (cg.cuh) when it
// has dropped by RELIABLE_DELTA since the last one, or when the float solver has stopped.
constexpr double RELIABLE_DELTA = 0.1;
constexpr double MIXED_TOL_F32 = 1e-5;     // relative recurrence residual asked of the float multi-shift phase

int mixed_solve_one(lqcd_ctx* c, const double* b, double sigma, double tol, double* x, bool have_guess, double bb,
                    int* iters_out, int* updates_out, double* rel_out) {
    int rc;
    PrecBufs<float>& F = bufs<float>(c);
    PrecBufs<double>& D = bufs<double>(c);
    const size_t n = c->Vh * 3;
    const int m = block_len(c);
    const double2* b2 = (const double2*)b;
    double2* x2 = (double2*)x;
    double2* ax = D.stage_x[0];           // (A + sigma) x
    float2* r0 = F.stage_b;               // float copy of the starting residual
    float2* y = F.stage_x[0];             // float partial solution since the last reliable update

    // device state of a single-shift float solve; the starting vector is the (true) starting residual
    CgState* h = c->st_host;
    memset(h, 0, sizeof(CgState));
    h->nshift = 1;
    h->i0 = 0;
    h->max_iter = c->max_iter;
    h->c0 = c->mass * c->mass + sigma;
    h->x[0] = (void*)y;
    h->p[0] = (void*)F.p;
    h->blk_m = m;
    for (int l = 0; l < m; ++l) h->hist[l] = (void*)F.hist[l];
    h->defer_base = defer_base(c);
    h->p_keep = (void*)F.p_keep;
    h->b_src = (const void*)r0;
    CU(cudaMemcpyAsync(c->st_dev, h, sizeof(CgState), cudaMemcpyHostToDevice, c->stream));

    if (have_guess) {
        if ((rc = apply_mdagm<double>(c, (double*)ax, x, sigma))) return rc;
    } else {
        CU(cudaMemsetAsync(x, 0, n * sizeof(double2), c->stream));
    }
    mixed_residual_kernel<<<cg_grid(c), CG_BLOCK, 0, c->stream>>>(b2, have_guess ? ax : nullptr, r0, c->st_dev, c->partials,
                                                                c->red, n, 0, 0);
    ++c->launches;
    CU(cudaMemcpyAsync(c->red_host, c->red, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    double rr_true = c->red_host[0];
    const double target = tol * tol * bb;
    *iters_out = 0;
    *updates_out = 0;
    *rel_out = std::sqrt(rr_true / bb);
    if (rr_true <= target) return LQCD_OK;

    CU(cudaMemsetAsync(y, 0, n * sizeof(float2), c->stream));       // should the float solver stop before its first sweep
    // tol of the float solver is relative to ITS source (the starting residual): same absolute target
    cg_init_kernel<float><<<cg_grid(c), CG_BLOCK, 0, c->stream>>>(r0, F.hist[m - 1], c->st_dev, c->partials, n,
                                                                 tol * std::sqrt(bb / rr_true));
    ++c->launches;
    CU(cudaGetLastError());

    const int ce = check_every(c);
    const bool use_graph = c->use_graph && c->stream != nullptr && c->stream != cudaStreamLegacy;
    if (use_graph && (F.graph_iters != ce || F.graph_block != m)) {
        if ((rc = build_graph<float>(c, ce, 0))) return rc;
    }
    double maxrr = rr_true;
    const long max_batches = (long)c->max_iter / ce + 3;
    for (long batch = 0; batch < max_batches; ++batch) {
        if (use_graph) {
            CU(cudaGraphLaunch(F.graph_exec, c->stream));
            c->launches += F.graph_launches;
        } else {
            for (int i = 0; i < ce; ++i)
                if ((rc = launch_cg_iteration<float>(c, i % m))) return rc;
            CU(cudaGetLastError());
        }
        // the head of the state: rr, ..., iter, stop, status
        CU(cudaMemcpyAsync(h, c->st_dev, offsetof(CgState, ticket), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        if (h->status == LQCD_EBREAKDOWN) return fail(c, LQCD_EBREAKDOWN, "<p,Ap> = %g at iteration %d", h->pAp, h->iter);
        if (h->rr > maxrr) maxrr = h->rr;
        if (!h->stop && !(h->rr < RELIABLE_DELTA * RELIABLE_DELTA * maxrr)) continue;

        // reliable update: x += y, y = 0, r <- b - (A + sigma) x in double, p keeps its direction
        mixed_accumulate_kernel<<<cg_grid(c), CG_BLOCK, 0, c->stream>>>(x2, y, n);
        ++c->launches;
        if ((rc = apply_mdagm<double>(c, (double*)ax, x, sigma))) return rc;
        // every batch starts at ring position 0 (a batch is a whole number of blocks, and a stop inside a block closes
        // it), i.e. its first iteration reads the residual from slot m-1 whatever slot the recurrence wrote last
        const int resume = (h->stop && h->status == 0) ? 1 : 0;
        mixed_residual_kernel<<<cg_grid(c), CG_BLOCK, 0, c->stream>>>(b2, ax, F.hist[m - 1], c->st_dev, c->partials, c->red, n,
                                                                    1, resume);
        ++c->launches;
        CU(cudaMemcpyAsync(c->red_host, c->red, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        rr_true = c->red_host[0];
        maxrr = rr_true;
        ++*updates_out;
        *iters_out = h->iter;
        *rel_out = std::sqrt(rr_true / bb);
        if (rr_true <= target) return LQCD_OK;
        if (h->stop && h->status == LQCD_ENOCONV)
            return fail(c, LQCD_ENOCONV, "no convergence in %d iterations, |r|/|b| = %.3e", h->iter, *rel_out);
    }
    return fail(c, LQCD_ENOCONV, "no convergence within the iteration cap, |r|/|b| = %.3e", *rel_out);
}

// Multi-shift front end: one float multi-shift solve brings every system to a loose tolerance, then each system is
// refined on its own (the shifted systems cannot share reliable updates: replacing r breaks r_i = zeta_i r).
int solve_mixed(lqcd_ctx* c, const double* b_even, const double* shifts, int nshift, double tol, double* const* x) {
    if (!c) return LQCD_EINVAL;
    if (!b_even || !shifts || !x) return fail(c, LQCD_EINVAL, "NULL argument");
    if (nshift < 1 || nshift > LQCD_MAX_SHIFTS) return fail(c, LQCD_EINVAL, "nshift must be in [1, %d]", LQCD_MAX_SHIFTS);
    if (!(tol > 0.0) || !std::isfinite(tol)) return fail(c, LQCD_EINVAL, "tol must be positive");
    for (int i = 0; i < nshift; ++i) {
        if (!(shifts[i] >= 0.0) || !std::isfinite(shifts[i])) return fail(c, LQCD_EINVAL, "shift %d must be >= 0", i);
        if (!x[i] || (const double*)x[i] == b_even) return fail(c, LQCD_EINVAL, "x[%d] is NULL or aliases b", i);
        for (int j = 0; j < i; ++j)
            if (x[j] == x[i]) return fail(c, LQCD_EINVAL, "x[%d] aliases x[%d]", i, j);
    }
    if (c->slab) return fail(c, LQCD_EINVAL, "the mixed-precision solver is not available on a slab context");
    int rc;
    if ((rc = check_ctx_gauge<double>(c)) || (rc = check_ctx_gauge<float>(c))) return rc;
    if ((rc = ensure_solver<float>(c, nshift)) || (rc = ensure_tmp<double>(c))) return rc;
    if ((rc = ensure_stage<float>(c, nshift)) || (rc = ensure_stage<double>(c, 1))) return rc;
    PrecBufs<float>& F = bufs<float>(c);
    PrecBufs<double>& D = bufs<double>(c);
    const size_t n = c->Vh * 3;
    const int cgrid = cg_grid(c);
    cudaEvent_t t0 = c->ev_m0, t1 = c->ev_m1;
    CU(cudaEventRecord(t0, c->stream));

    // |b|^2 in double (the residual kernel with nothing subtracted), and the float copy of b
    CU(cudaMemsetAsync(c->st_dev, 0, sizeof(CgState), c->stream));
    mixed_residual_kernel<<<cgrid, CG_BLOCK, 0, c->stream>>>((const double2*)b_even, nullptr, F.stage_b, c->st_dev, c->partials,
                                                           c->red, n, 0, 0);
    ++c->launches;
    CU(cudaMemcpyAsync(c->red_host, c->red, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    const double bb = c->red_host[0];
    int total_iters = 0, total_updates = 0;
    double worst = 0.0;
    c->last_nshift = nshift;
    if (bb == 0.0) {
        for (int i = 0; i < nshift; ++i) CU(cudaMemsetAsync(x[i], 0, n * sizeof(double2), c->stream));
        for (int i = 0; i < nshift; ++i) c->last_freeze[i] = 0;
    } else {
        bool guess = false;
        if (nshift > 1) {
            // phase 1: every system at once in single precision, to what single precision can deliver
            const double tol1 = tol > MIXED_TOL_F32 ? tol : MIXED_TOL_F32;
            float* xf[LQCD_MAX_SHIFTS];
            for (int i = 0; i < nshift; ++i) xf[i] = (float*)F.stage_x[i];
            rc = solve<float>(c, (const float*)F.stage_b, shifts, nshift, tol1, xf, nullptr, 0.0, nullptr);
            if (rc != LQCD_OK && rc != LQCD_ENOCONV) return rc;
            total_iters += c->last_iters;
            for (int i = 0; i < nshift; ++i) {
                convert_vector_kernel<double, float><<<cgrid, 256, 0, c->stream>>>(F.stage_x[i], (double2*)x[i], n);
                ++c->launches;
            }
            guess = true;
        }
        // phase 2: each system to the double-precision tolerance
        for (int i = 0; i < nshift; ++i) {
            int it = 0, up = 0;
            double rel = 0.0;
            rc = mixed_solve_one(c, b_even, shifts[i], tol, x[i], guess, bb, &it, &up, &rel);
            total_iters += it;
            total_updates += up;
            c->last_freeze[i] = it;
            if (rel > worst) worst = rel;
            if (rc != LQCD_OK) {
                c->last_iters = total_iters;
                c->last_rel = worst;
                c->last_updates = total_updates;
                return rc;
            }
        }
    }
    CU(cudaEventRecord(t1, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    CU(cudaEventElapsedTime(&c->last_ms, t0, t1));
    c->last_iters = total_iters;
    c->last_rel = worst;
    c->last_updates = total_updates;
    c->last_i0 = 0;
    (void)D;
    return LQCD_OK;
}

template <typename T>
int pack_unpack(lqcd_ctx* c, int parity, const T* in, T* out, bool pack) {
    if (!c) return LQCD_EINVAL;
    if (!in || !out || (parity != 0 && parity != 1)) return fail(c, LQCD_EINVAL, "bad argument");
    const int grid = (int)((c->Vh + 255) / 256);
    if (pack)
        pack_vector_kernel<T><<<grid, 256, 0, c->stream>>>(c->g, parity, (const V2<T>*)in, (V2<T>*)out);
    else
        unpack_vector_kernel<T><<<grid, 256, 0, c->stream>>>(c->g, parity, (const V2<T>*)in, (V2<T>*)out);
    ++c->launches;
    CU(cudaGetLastError());
    return LQCD_OK;
}

}  // namespace

// ---- lqcd_mdagm_static: the Eq. 2 operator for callers that must not allocate device memory (include/lqcd.h) -----
// lqcd_mdagm keeps the odd-parity intermediate t = D_oe v in a buffer it allocates on first use.  Here that
// intermediate lives in the array below, which is part of the library's image: the CUDA runtime places one copy of it
// on every device that loads this module and keeps it until the process exits, whether or not the entry point is
// ever called.  LQCD_STATIC_MAX_VH sites per parity x 3 colours x 16 bytes = 3 MiB.
static __device__ __align__(256) double2 g_static_t[3 * (size_t)LQCD_STATIC_MAX_VH];

namespace {

// In host code `g_static_t` is only the handle under which the runtime knows the array -- it is not something a
// kernel can dereference.  The address that kernels can use differs from device to device and is asked for once
// per device, with that device current.
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
double2* g_static_addr[STATIC_MAX_DEVICES] = {};

int static_scratch(lqcd_ctx* c, double2** out) {
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev != c->device)
        return fail(c, LQCD_EINVAL, "lqcd_mdagm_static: the context belongs to device %d but device %d is current", c->device,
                    dev);
    if (dev < 0 || dev >= STATIC_MAX_DEVICES)
        return fail(c, LQCD_EINVAL, "lqcd_mdagm_static: device ordinal %d not supported (< %d)", dev, STATIC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_addr[dev]) {
        void* p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_static_t));
        if (!p) return fail(c, LQCD_ECUDA, "lqcd_mdagm_static: cudaGetSymbolAddress gave a NULL address");
        g_static_addr[dev] = (double2*)p;
    }
    *out = g_static_addr[dev];
    return LQCD_OK;
}

}  // namespace

extern "C" {

int lqcd_comm_abort(lqcd_ctx* c) {
    if (!c) return LQCD_EINVAL;
    if (!c->slab) return fail(c, LQCD_EINVAL, "not a slab context");
    if (c->p2p.active) lqcd_p2p::poison(&c->p2p, true);
    return LQCD_OK;
}

int lqcd_mdagm_static(lqcd_ctx* c, double* out_even, const double* in_even, double sigma) {
    if (!c) return LQCD_EINVAL;
    if (!out_even || !in_even) return fail(c, LQCD_EINVAL, "NULL vector");
    if (out_even == in_even) return fail(c, LQCD_EINVAL, "in and out must not alias");
    if (c->slab) return fail(c, LQCD_EINVAL, "lqcd_mdagm_static: whole-lattice contexts only (a slab needs halo buffers)");
    if (c->Vh > (size_t)LQCD_STATIC_MAX_VH)
        return fail(c, LQCD_EINVAL, "lqcd_mdagm_static: the lattice has %zu sites per parity, the built-in buffer holds at "
                    "most %d (LQCD_STATIC_MAX_VH); use lqcd_mdagm", c->Vh, (int)LQCD_STATIC_MAX_VH);
    int rc;
    if ((rc = check_ctx_gauge<double>(c))) return rc;
    double2* t = nullptr;
    if ((rc = static_scratch(c, &t))) return rc;
    // the same two launches as lqcd_mdagm; the first one writes every odd site of t, so nothing of an earlier call
    // is read and nothing has to be cleared
    launch_dslash<double>(c, 0, t, (const double2*)in_even, 1, nullptr, 0.0, 0);
    launch_dslash<double>(c, 2, (double2*)out_even, t, 0, (const double2*)in_even, c->mass * c->mass + sigma, 0);
    CU(cudaGetLastError());
    return LQCD_OK;
}

int lqcd_doe(lqcd_ctx* c, double* out_odd, const double* in_even) { return apply_d<double>(c, out_odd, in_even, 1); }
int lqcd_deo(lqcd_ctx* c, double* out_even, const double* in_odd) { return apply_d<double>(c, out_even, in_odd, 0); }
int lqcd_doe_host(lqcd_ctx* c, double* out_odd, const double* in_even) { return apply_d_host<double>(c, out_odd, in_even, 1); }
int lqcd_deo_host(lqcd_ctx* c, double* out_even, const double* in_odd) { return apply_d_host<double>(c, out_even, in_odd, 0); }
int lqcd_mdagm(lqcd_ctx* c, double* out_even, const double* in_even, double sigma) {
    return apply_mdagm<double>(c, out_even, in_even, sigma);
}

int lqcd_doe_f32(lqcd_ctx* c, float* out_odd, const float* in_even) { return apply_d<float>(c, out_odd, in_even, 1); }
int lqcd_deo_f32(lqcd_ctx* c, float* out_even, const float* in_odd) { return apply_d<float>(c, out_even, in_odd, 0); }
int lqcd_doe_f32_host(lqcd_ctx* c, float* out_odd, const float* in_even) { return apply_d_host<float>(c, out_odd, in_even, 1); }
int lqcd_deo_f32_host(lqcd_ctx* c, float* out_even, const float* in_odd) { return apply_d_host<float>(c, out_even, in_odd, 0); }
int lqcd_mdagm_f32(lqcd_ctx* c, float* out_even, const float* in_even, double sigma) {
    return apply_mdagm<float>(c, out_even, in_even, sigma);
}

int lqcd_mshift_cg(lqcd_ctx* c, const double* b_even, const double* shifts, int nshift, double tol, double* const* x) {
    if (c && !x) return fail(c, LQCD_EINVAL, "NULL argument");
    return solve<double>(c, b_even, shifts, nshift, tol, x, nullptr, 0.0, nullptr);
}
int lqcd_mshift_cg_host(lqcd_ctx* c, const double* b_even, const double* shifts, int nshift, double tol, double* const* x) {
    if (c && !x) return fail(c, LQCD_EINVAL, "NULL argument");
    return solve_host<double>(c, b_even, shifts, nshift, tol, x, nullptr, 0.0, nullptr);
}
int lqcd_mshift_cg_f32(lqcd_ctx* c, const float* b_even, const double* shifts, int nshift, double tol, float* const* x) {
    if (c && !x) return fail(c, LQCD_EINVAL, "NULL argument");
    return solve<float>(c, b_even, shifts, nshift, tol, x, nullptr, 0.0, nullptr);
}
int lqcd_mshift_cg_f32_host(lqcd_ctx* c, const float* b_even, const double* shifts, int nshift, double tol, float* const* x) {
    if (c && !x) return fail(c, LQCD_EINVAL, "NULL argument");
    return solve_host<float>(c, b_even, shifts, nshift, tol, x, nullptr, 0.0, nullptr);
}

int lqcd_mshift_cg_mixed(lqcd_ctx* c, const double* b_even, const double* shifts, int nshift, double tol, double* const* x) {
    return solve_mixed(c, b_even, shifts, nshift, tol, x);
}

int lqcd_rational_apply(lqcd_ctx* c, const double* b_even, double alpha0, const double* alpha, const double* shifts,
                        int nshift, double tol, double* y_even) {
    if (c && (!y_even || !alpha)) return fail(c, LQCD_EINVAL, "NULL argument");
    return solve<double>(c, b_even, shifts, nshift, tol, nullptr, y_even, alpha0, alpha);
}
int lqcd_rational_apply_host(lqcd_ctx* c, const double* b_even, double alpha0, const double* alpha,
                             const double* shifts, int nshift, double tol, double* y_even) {
    if (c && (!y_even || !alpha)) return fail(c, LQCD_EINVAL, "NULL argument");
    return solve_host<double>(c, b_even, shifts, nshift, tol, nullptr, y_even, alpha0, alpha);
}
int lqcd_rational_apply_f32(lqcd_ctx* c, const float* b_even, double alpha0, const double* alpha, const double* shifts,
                            int nshift, double tol, float* y_even) {
    if (c && (!y_even || !alpha)) return fail(c, LQCD_EINVAL, "NULL argument");
    return solve<float>(c, b_even, shifts, nshift, tol, nullptr, y_even, alpha0, alpha);
}

int lqcd_get_stat(const lqcd_ctx* c, int key, int idx, double* out) {
    if (!c || !out) return LQCD_EINVAL;
    switch (key) {
        case LQCD_STAT_ITERS: *out = c->last_iters; break;
        case LQCD_STAT_REL_RES: *out = c->last_rel; break;
        case LQCD_STAT_FREEZE_ITER:
            if (idx < 0 || idx >= c->last_nshift) return LQCD_EINVAL;
            *out = c->last_freeze[idx];
            break;
        case LQCD_STAT_BASE_SHIFT: *out = c->last_i0; break;
        case LQCD_STAT_GPU_LAUNCHES: *out = (double)c->launches; break;
        case LQCD_STAT_SOLVE_MS: *out = c->last_ms; break;
        case LQCD_STAT_RELIABLE_UPDATES: *out = c->last_updates; break;
        case LQCD_STAT_GRAPH_REPLAYS: *out = c->last_replays; break;
        case LQCD_STAT_SOLVER_PATH: *out = c->last_path; break;
        default: return LQCD_EINVAL;
    }
    return LQCD_OK;
}

int lqcd_pack_vector(lqcd_ctx* c, int parity, const double* site_field, double* parity_vector) {
    return pack_unpack<double>(c, parity, site_field, parity_vector, true);
}
int lqcd_unpack_vector(lqcd_ctx* c, int parity, const double* parity_vector, double* site_field) {
    return pack_unpack<double>(c, parity, parity_vector, site_field, false);
}
int lqcd_pack_vector_f32(lqcd_ctx* c, int parity, const float* site_field, float* parity_vector) {
    return pack_unpack<float>(c, parity, site_field, parity_vector, true);
}
int lqcd_unpack_vector_f32(lqcd_ctx* c, int parity, const float* parity_vector, float* site_field) {
    return pack_unpack<float>(c, parity, parity_vector, site_field, false);
}

}  // extern "C"
