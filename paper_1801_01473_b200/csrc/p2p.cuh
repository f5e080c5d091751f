// p2p.cuh -- the two exchange steps of the slab-decomposed path over peer-mapped memory (NVLink 5 / NVSwitch
// between the GPUs of a node; the paper: "CUDA-aware MPI ... CUDA inter-process communication between GPUs attached
// to the same host").  No NCCL kernel, no staging buffer:
//
//   * every rank owns ONE device allocation, its WINDOW: a header of flag words and all-reduce slots, then four face
//     buffers ([from rank-1 | from rank+1] x two generations).  The window is exported with cudaIpcGetMemHandle; the
//     handles travel once over the caller's channel (lqcd_p2p_export / lqcd_comm_init_p2p), and every rank maps every
//     other rank's window (cudaIpcOpenMemHandle enables peer access over NVLink);
//   * face exchange number s (one counter per rank, the same on all of them), generation g = s&1: the sender WRITES its
//     two faces straight into the neighbours' face buffers of generation g -- strided copies or the stores of the
//     pack kernel, from the vector itself -- then sets the neighbours' `arrived[side][g]` words to 1 with a stream
//     memory operation (cuStreamWriteValue32, ordered after the copies), waits for its own two `arrived[.][g]` words
//     (cuStreamWaitValue32 on LOCAL memory).  The border launch reads the halo in place, in the window, and clears
//     the two words;
//   * no flow control is needed beyond the two generations: a rank that sends face s has received face s-1 from that
//     neighbour, which the neighbour sent (stream order) after it had cleared its flags of s-2 and launched the
//     kernel that consumed ITS halo of s-2, the last tenant of the buffer and flag now being overwritten;
//   * all-reduce of the scalar products, generation g = q&1 of all-reduce number q: the rank's value is stored into
//     slot [g][rank] of every rank's window (its own included) and then, after a system-wide fence, 1 into their
//     `red_arrived[g][rank]` words (peer_push: by the one-block kernel that sums the rank's block partials, or by
//     p2p_push_kernel); nranks stream waits on the local words; one kernel adds the slots in rank order -- every
//     rank holds the same bits (R8) --, clears the words and runs the scalar step of the CG.  The same
//     two-generation argument applies.
//
// Nothing here spins inside a kernel: every wait is a stream memory operation on the waiting rank's own memory, so
// several ranks may share one GPU (tests) without any kernel of one waiting for a kernel of another.
// Every value written or waited for is the constant 0 or 1 and every address depends only on the generation, so the
// operations of a CG iteration (two exchanges, two all-reduces: the generations come round) CAN be captured into a
// CUDA graph; that was built and measured (correct, and slower than plain launches at 16^4, 32^4 and 48^4: a memory
// operation node costs more than the launch it saves), so the library launches the iteration plainly (graph_safe = 0).
#ifndef LQCD_P2P_CUH
#define LQCD_P2P_CUH

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>
#include <unistd.h>

#include "lqcd_internal.cuh"

namespace lqcd_p2p {

constexpr int MAX_RANKS = LQCD_P2P_MAX_RANKS;
constexpr int RED_MAX = LQCD_P2P_RED_MAX;
constexpr size_t HDR_BYTES = 4096;

struct Header {                            // start of every window
    unsigned int arrived[2][2];            // [side: 0 = from rank-1, 1 = from rank+1][generation]: 1 = that face is complete
    unsigned int pad[12];
    unsigned int red_arrived[2][MAX_RANKS];   // [generation][rank]: 1 = that rank's contribution is in its slot
    double red[2][MAX_RANKS][RED_MAX];     // [generation][rank][value]
    PeerPush push[2];                      // this rank's targets of generation 0 / 1 (addresses as mapped HERE)
};
static_assert(sizeof(Header) <= HDR_BYTES, "window header");

// what travels between the ranks (LQCD_P2P_HANDLE_BYTES of include/lqcd.h)
struct Blob {
    cudaIpcMemHandle_t ipc;                // 64 bytes
    long long pid;                         // process_tag() of the exporter: its pid and a number drawn once per process
    unsigned long long ptr;                // the window in the exporting process (used when it is this process)
    unsigned long long cap;
    int device;
    int rank;
};
static_assert(sizeof(Blob) == 96, "LQCD_P2P_HANDLE_BYTES");

typedef CUresult (*mem_op32_fn)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);

struct Transport {
    bool active = false;
    int rank = 0, nranks = 1, device = 0;
    char* win[MAX_RANKS] = {};             // every rank's window as mapped in this process; win[rank] is mine
    bool opened[MAX_RANKS] = {};           // mapped with cudaIpcOpenMemHandle (to be closed)
    size_t cap = 0;                        // bytes of one face buffer
    unsigned int seq = 0, rseq = 0;        // exchanges / all-reduces issued so far (only their parity matters)
    mem_op32_fn wait32 = nullptr, write32 = nullptr;
    bool kernel_signal = false;            // remote arrival words are set by a one-thread kernel, not by cuStreamWriteValue32
    bool dead = false;                     // an operation failed after connect: every later one is refused at once
    const char* error = "";

    Header* hdr(int r) const { return (Header*)win[r]; }
    Header* mine() const { return (Header*)win[rank]; }
    // face buffer of rank r: side 0 = halo below its slab (filled by r-1), 1 = above (filled by r+1)
    char* face(int r, int side, unsigned int g) const { return win[r] + HDR_BYTES + ((size_t)side * 2 + (g & 1)) * cap; }
    int dn() const { return (rank + nranks - 1) % nranks; }
    int up() const { return (rank + 1) % nranks; }
};

inline size_t window_bytes(size_t cap) { return HDR_BYTES + 4 * cap; }

// A failure after connect() leaves this rank's exchange counters (seq, rseq) out of step with its peers', and
// possibly half an exchange enqueued: nothing further can be matched, so the transport is dead from then on and
// keeps the text of the first failure.
inline int fail(Transport* t, const char* why) {
    if (!t->dead) t->error = why;
    if (t->active) t->dead = true;
    cudaGetLastError();
    return -1;
}
inline bool usable(const Transport* t) { return t->active && !t->dead; }

// Two ranks are "the same process" (and may use each other's device pointers as they are) only if pid AND a number
// drawn once per process agree: ranks in different PID namespaces of one node (a container each) can have equal pids.
inline long long process_tag() {
    static long long tag = 0;
    if (!tag) {
        unsigned int nonce = 0;
        FILE* f = fopen("/dev/urandom", "rb");
        if (f) {
            if (fread(&nonce, sizeof(nonce), 1, f) != 1) nonce = 0;
            fclose(f);
        }
        if (!nonce) nonce = (unsigned int)((uintptr_t)&tag & 0xffffffffu) ^ (unsigned int)time(nullptr);
        tag = ((long long)(unsigned int)getpid() << 32) | (long long)(nonce | 1u);
    }
    return tag;
}

// allocate this rank's window and describe it
inline int create_window(Transport* t, int rank, int nranks, size_t cap, Blob* out) {
    if (nranks > MAX_RANKS) return fail(t, "more ranks than the peer-memory transport handles");
    if (t->win[rank]) return fail(t, "window already exported");
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuStreamWaitValue32", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn)
        return fail(t, "cuStreamWaitValue32 not available");
    t->wait32 = (mem_op32_fn)fn;
    if (cudaGetDriverEntryPoint("cuStreamWriteValue32", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn)
        return fail(t, "cuStreamWriteValue32 not available");
    t->write32 = (mem_op32_fn)fn;
    t->rank = rank;
    t->nranks = nranks;
    const char* ks = getenv("LQCD_P2P_KERNEL_SIGNAL");       // tests: take the fall-back of signal_wait from the start
    t->kernel_signal = ks && ks[0] == '1';
    t->cap = (cap + 255) / 256 * 256;
    if (cudaGetDevice(&t->device) != cudaSuccess) return fail(t, "cudaGetDevice");
    void* w = nullptr;
    if (cudaMalloc(&w, window_bytes(t->cap)) != cudaSuccess) return fail(t, "cudaMalloc of the window");
    if (cudaMemset(w, 0, HDR_BYTES) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) {
        cudaFree(w);
        return fail(t, "clearing the window");
    }
    t->win[rank] = (char*)w;
    memset(out, 0, sizeof(Blob));
    if (cudaIpcGetMemHandle(&out->ipc, w) != cudaSuccess) cudaGetLastError();   // ranks of one process need no handle
    out->pid = process_tag();
    out->ptr = (unsigned long long)(uintptr_t)w;
    out->cap = t->cap;
    out->device = t->device;
    out->rank = rank;
    return 0;
}

// map every rank's window; write the push targets of both generations into my header
inline int connect(Transport* t, const Blob* blobs) {
    if (!t->win[t->rank]) return fail(t, "lqcd_p2p_export first");
    for (int r = 0; r < t->nranks; ++r) {
        const Blob& b = blobs[r];
        if (b.rank != r || b.cap != t->cap) return fail(t, "handle table does not match this lattice / rank order");
        if (r == t->rank) continue;
        if (b.pid == process_tag()) {
            // another context of this process: its pointer is valid here (checked); peer access if it sits on another
            // device
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, (const void*)(uintptr_t)b.ptr) != cudaSuccess ||
                at.type != cudaMemoryTypeDevice || at.device != b.device)
                return fail(t, "a handle claims to come from this process but its window is not device memory here");
            if (b.device != t->device) {
                const cudaError_t e = cudaDeviceEnablePeerAccess(b.device, 0);
                if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) return fail(t, "no peer access to a rank of this process");
                cudaGetLastError();
            }
            t->win[r] = (char*)(uintptr_t)b.ptr;
        } else {
            void* p = nullptr;
            if (cudaIpcOpenMemHandle(&p, b.ipc, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess)
                return fail(t, "cudaIpcOpenMemHandle failed (ranks must be on GPUs of one node with peer access)");
            t->win[r] = (char*)p;
            t->opened[r] = true;
        }
    }
    PeerPush push[2];
    memset(push, 0, sizeof(push));
    for (int g = 0; g < 2; ++g) {
        push[g].nranks = t->nranks;
        for (int r = 0; r < t->nranks; ++r) {
            push[g].slot[r] = &t->hdr(r)->red[g][t->rank][0];
            push[g].flag[r] = &t->hdr(r)->red_arrived[g][t->rank];
        }
    }
    if (cudaMemcpy(t->mine()->push, push, sizeof(push), cudaMemcpyHostToDevice) != cudaSuccess)
        return fail(t, "writing the push targets");
    t->active = true;
    return 0;
}

// Release every rank that waits, or will wait, for something from this rank: LQCD_P2P_POISON into the arrival words this
// rank is the writer of -- the face words of its two neighbours and its own entry of every rank's all-reduce words, both
// generations.  Their stream waits complete, the kernels behind them find the mark and end the solve with LQCD_ECOMM
// (cg.cuh, dslash.cuh), and every rank that returns LQCD_ECOMM does the same for ITS peers, so the release spreads to
// ranks that were waiting for somebody else.  self = true (a rank that waited too long for a peer that may be gone
// without a word): also all of this rank's own words, so that its own streams drain.
// Plain 4-byte copies on a stream of their own: the rank's other streams may be the ones that are stuck.
inline void poison(Transport* t, bool self) {
    if (!t->win[t->rank]) return;
    t->dead = true;
    if (!*t->error) t->error = "aborted";
    cudaStream_t s = nullptr;
    if (cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError();
        return;
    }
    static const unsigned int mark = LQCD_P2P_POISON;
    auto put = [&](unsigned int* w) { cudaMemcpyAsync(w, &mark, sizeof(mark), cudaMemcpyDefault, s); };
    for (int g = 0; g < 2; ++g) {
        if (t->win[t->dn()]) put(&t->hdr(t->dn())->arrived[1][g]);
        if (t->win[t->up()]) put(&t->hdr(t->up())->arrived[0][g]);
        for (int r = 0; r < t->nranks; ++r)
            if (t->win[r]) put(&t->hdr(r)->red_arrived[g][t->rank]);
        if (self) {
            put(&t->mine()->arrived[0][g]);
            put(&t->mine()->arrived[1][g]);
            for (int r = 0; r < t->nranks; ++r) put(&t->mine()->red_arrived[g][r]);
        }
    }
    cudaStreamSynchronize(s);
    cudaStreamDestroy(s);
    cudaGetLastError();
}

inline void destroy(Transport* t) {
    for (int r = 0; r < t->nranks; ++r)
        if (t->opened[r]) cudaIpcCloseMemHandle(t->win[r]);
    if (t->win[t->rank]) cudaFree(t->win[t->rank]);
    for (int r = 0; r < MAX_RANKS; ++r) {
        t->win[r] = nullptr;
        t->opened[r] = false;
    }
    t->active = false;
    cudaGetLastError();
}

inline CUdeviceptr dptr(const void* p) { return (CUdeviceptr)(uintptr_t)p; }

// Where the faces of the NEXT exchange go and arrive: the sender writes its lowest slice to dst_dn and its highest to
// dst_up (peer memory); recv_lo / recv_hi are this rank's own halo buffers of that exchange.
struct Slots {
    void *dst_dn, *dst_up, *recv_lo, *recv_hi;
};
inline Slots begin(Transport* t) {
    const unsigned int g = ++t->seq & 1;
    Slots o;
    o.dst_dn = t->face(t->dn(), 1, g);       // my lowest slice is the halo ABOVE the slab of rank-1
    o.dst_up = t->face(t->up(), 0, g);       // my highest slice is the halo BELOW the slab of rank+1
    o.recv_lo = t->face(t->rank, 0, g);
    o.recv_hi = t->face(t->rank, 1, g);
    return o;
}
// after the writes to dst_dn / dst_up have been enqueued on `stream`: tell the neighbours, wait for mine, clear
// (clear = false: the kernel that consumes the halos clears the two words itself, clear_words())
inline void clear_words(Transport* t, unsigned int** w0, unsigned int** w1) {
    *w0 = &t->mine()->arrived[0][t->seq & 1];
    *w1 = &t->mine()->arrived[1][t->seq & 1];
}
// the two arrival words of a face exchange, set from a kernel: the fall-back when the driver refuses a stream memory
// operation on a peer-mapped address (stores from kernels are what peer access is for)
__global__ void p2p_signal_kernel(unsigned int* a, unsigned int* b) {
    __threadfence_system();
    *(volatile unsigned int*)a = 1u;
    *(volatile unsigned int*)b = 1u;
}
// the two arrival words back to 0 for their next use, except a word that holds the mark of a rank that gave up
__global__ void p2p_clear_kernel(unsigned int* a, unsigned int* b) {
    unsigned int* w = threadIdx.x ? b : a;
    if (*(volatile unsigned int*)w != LQCD_P2P_POISON) *w = 0u;
}
inline int signal_wait(Transport* t, cudaStream_t stream, bool clear = true) {
    const unsigned int g = t->seq & 1;
    CUstream cs = (CUstream)stream;
    unsigned int* mine[2] = {&t->mine()->arrived[0][g], &t->mine()->arrived[1][g]};
    unsigned int* dn = &t->hdr(t->dn())->arrived[1][g];
    unsigned int* up = &t->hdr(t->up())->arrived[0][g];
    if (!t->kernel_signal && t->write32(cs, dptr(dn), 1u, CU_STREAM_WRITE_VALUE_DEFAULT) != CUDA_SUCCESS) {
        cudaGetLastError();
        t->kernel_signal = true;               // nothing has been signalled yet: both words go by kernel from now on
    }
    if (t->kernel_signal) {
        p2p_signal_kernel<<<1, 1, 0, stream>>>(dn, up);
        if (cudaGetLastError() != cudaSuccess) return fail(t, "signalling a neighbour's window failed");
    } else if (t->write32(cs, dptr(up), 1u, CU_STREAM_WRITE_VALUE_DEFAULT) != CUDA_SUCCESS) {
        return fail(t, "cuStreamWriteValue32 on a neighbour's window failed");
    }
    for (int side = 0; side < 2; ++side)
        if (t->wait32(cs, dptr(mine[side]), 1u, CU_STREAM_WAIT_VALUE_GEQ) != CUDA_SUCCESS) return fail(t, "cuStreamWaitValue32 failed");
    if (clear) {
        p2p_clear_kernel<<<1, 2, 0, stream>>>(mine[0], mine[1]);
        if (cudaGetLastError() != cudaSuccess) return fail(t, "clearing the arrival words failed");
    }
    return 0;
}

// lqcd_comm_ops::exchange for arbitrary buffers (the one-time link faces): through the window, then out of it
inline int exchange(void* user, const void* send_lo, const void* send_hi, void* recv_lo, void* recv_hi, size_t bytes,
                    void* stream) {
    Transport* t = (Transport*)user;
    if (t->dead) return -1;
    if (!t->active) return fail(t, "transport not connected");
    if (bytes > t->cap) return fail(t, "message larger than a face buffer of the window");
    cudaStream_t s = (cudaStream_t)stream;
    const Slots o = begin(t);
    if (cudaMemcpyAsync(o.dst_dn, send_lo, bytes, cudaMemcpyDefault, s) != cudaSuccess ||
        cudaMemcpyAsync(o.dst_up, send_hi, bytes, cudaMemcpyDefault, s) != cudaSuccess)
        return fail(t, "copy into a neighbour's window failed");
    if (signal_wait(t, s)) return -1;
    if (cudaMemcpyAsync(recv_lo, o.recv_lo, bytes, cudaMemcpyDeviceToDevice, s) != cudaSuccess ||
        cudaMemcpyAsync(recv_hi, o.recv_hi, bytes, cudaMemcpyDeviceToDevice, s) != cudaSuccess)
        return fail(t, "copy out of the window failed");
    return 0;
}

// ---- all-reduce.  Three steps: push (by the producer of the value, or p2p_push_kernel), wait, sum + clear.
// reduce_begin opens all-reduce number ++rseq and returns the push targets of its generation (device memory).
inline const PeerPush* reduce_begin(Transport* t) { return &t->mine()->push[++t->rseq & 1]; }
inline int reduce_wait(Transport* t, cudaStream_t stream) {
    const unsigned int g = t->rseq & 1;
    for (int r = 0; r < t->nranks; ++r)
        if (t->wait32((CUstream)stream, dptr(&t->mine()->red_arrived[g][r]), 1u, CU_STREAM_WAIT_VALUE_GEQ) != CUDA_SUCCESS)
            return fail(t, "cuStreamWaitValue32 failed");
    return 0;
}
inline double* reduce_slots(Transport* t) { return &t->mine()->red[t->rseq & 1][0][0]; }
inline unsigned int* reduce_flags(Transport* t) { return &t->mine()->red_arrived[t->rseq & 1][0]; }

__global__ void __launch_bounds__(32) p2p_push_kernel(const PeerPush* __restrict__ d, const double* __restrict__ value, int n) {
    const int q = threadIdx.x;
    if (q >= d->nranks) return;
    for (int j = 0; j < n; ++j) ((volatile double*)d->slot[q])[j] = value[j];
    __threadfence_system();
    *(volatile unsigned int*)d->flag[q] = 1u;
}
// out[j] = sum over ranks, in rank order: the same bits on every rank; the flags are cleared for their next use
__global__ void __launch_bounds__(32) p2p_sum_kernel(const double* slots, unsigned int* flags, int nranks, int n,
                                                     double* __restrict__ out) {
    const int j = threadIdx.x;
    if (j < n) {
        double acc = 0.0;
        for (int r = 0; r < nranks; ++r) acc += __ldcv(slots + r * RED_MAX + j);
        out[j] = acc;
    }
    if (j < nranks && *(volatile unsigned int*)(flags + j) != LQCD_P2P_POISON) flags[j] = 0u;   // the mark of a rank that gave up stays
}

inline int allreduce_sum(void* user, double* dev_buf, int n, void* stream) {
    Transport* t = (Transport*)user;
    if (t->dead) return -1;
    if (!t->active) return fail(t, "transport not connected");
    if (n < 1 || n > RED_MAX) return fail(t, "all-reduce of more values than a slot holds");
    cudaStream_t s = (cudaStream_t)stream;
    p2p_push_kernel<<<1, 32, 0, s>>>(reduce_begin(t), dev_buf, n);
    if (reduce_wait(t, s)) return -1;
    p2p_sum_kernel<<<1, 32, 0, s>>>(reduce_slots(t), reduce_flags(t), t->nranks, n, dev_buf);
    if (cudaGetLastError() != cudaSuccess) return fail(t, "launch of the all-reduce kernels failed");
    return 0;
}

}  // namespace lqcd_p2p

#endif
