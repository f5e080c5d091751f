// comm.h -- the two exchange steps of the slab-decomposed path and their transports.
//
// The paper cuts the lattice along one direction and needs, per application of D_oe / D_eo, the faces of the
// input vector from the two neighbouring ranks, plus "global reductions" for the scalar products
// (Alg. 1).  Those are the only two communication steps of the path:
//     exchange       send my lowest time slice to rank-1 and my highest to rank+1 (periodic ring);
//                    receive rank-1's highest slice (-> recv_lo) and rank+1's lowest (-> recv_hi)
//     allreduce_sum  sum n doubles over all ranks, same bits on every rank
// A transport is a pair of functions (lqcd_comm_ops, include/lqcd.h).  Built in: NCCL (send/recv and all-reduce
// over NVLink 5 / NVSwitch), resolved with dlopen so that the library carries no link-time dependency and the
// NCCL already loaded by the host process (torch's) is the one used.  The Python binding supplies a second one
// on top of torch.distributed for tests (host-staged through gloo: several ranks may then share one GPU, none of
// their kernels ever waits on another rank).
#ifndef LQCD_COMM_H
#define LQCD_COMM_H

#include <cuda_runtime.h>
#include <dlfcn.h>
#include <stddef.h>
#include <string.h>

namespace lqcd_nccl {

// the part of NCCL's public C API that is used (restated from its documentation; values of the enums as in nccl.h)
typedef struct ncclComm* comm_t;
typedef struct { char internal[128]; } unique_id;
enum { kSuccess = 0 };
enum { kSum = 0 };
enum { kChar = 0, kFloat64 = 8 };

struct Api {
    void* handle = nullptr;
    int (*GetUniqueId)(unique_id*) = nullptr;
    int (*CommInitRank)(comm_t*, int, unique_id, int) = nullptr;
    int (*CommDestroy)(comm_t) = nullptr;
    int (*Send)(const void*, size_t, int, int, comm_t, cudaStream_t) = nullptr;
    int (*Recv)(void*, size_t, int, int, comm_t, cudaStream_t) = nullptr;
    int (*AllReduce)(const void*, void*, size_t, int, int, comm_t, cudaStream_t) = nullptr;
    int (*GroupStart)() = nullptr;
    int (*GroupEnd)() = nullptr;
    const char* (*GetErrorString)(int) = nullptr;
};

inline Api* api(const char** why) {
    static Api a;
    static bool tried = false;
    static const char* err = nullptr;
    if (!tried) {
        tried = true;
        a.handle = dlopen("libnccl.so.2", RTLD_NOW | RTLD_GLOBAL);
        if (!a.handle) a.handle = dlopen("libnccl.so", RTLD_NOW | RTLD_GLOBAL);
        if (!a.handle) {
            err = "libnccl.so.2 not found";
        } else {
#define LQCD_NCCL_SYM(field, name)                                        \
    *(void**)(&a.field) = dlsym(a.handle, name);                          \
    if (!a.field && !err) err = "NCCL symbol missing: " name;
            LQCD_NCCL_SYM(GetUniqueId, "ncclGetUniqueId")
            LQCD_NCCL_SYM(CommInitRank, "ncclCommInitRank")
            LQCD_NCCL_SYM(CommDestroy, "ncclCommDestroy")
            LQCD_NCCL_SYM(Send, "ncclSend")
            LQCD_NCCL_SYM(Recv, "ncclRecv")
            LQCD_NCCL_SYM(AllReduce, "ncclAllReduce")
            LQCD_NCCL_SYM(GroupStart, "ncclGroupStart")
            LQCD_NCCL_SYM(GroupEnd, "ncclGroupEnd")
            LQCD_NCCL_SYM(GetErrorString, "ncclGetErrorString")
#undef LQCD_NCCL_SYM
        }
    }
    if (why) *why = err;
    return err ? nullptr : &a;
}

struct Transport {
    comm_t comm = nullptr;
    int rank = 0, nranks = 1;
    int last_error = 0;
};

// lqcd_comm_ops::exchange over NCCL: four point-to-point operations in one group, enqueued on `stream`
inline int exchange(void* user, const void* send_lo, const void* send_hi, void* recv_lo, void* recv_hi, size_t bytes,
                    void* stream) {
    Transport* t = (Transport*)user;
    Api* a = api(nullptr);
    if (!a || !t->comm) return -1;
    const int dn = (t->rank + t->nranks - 1) % t->nranks, up = (t->rank + 1) % t->nranks;
    cudaStream_t s = (cudaStream_t)stream;
    // Operations between one pair of ranks are matched in the order they are issued.  With two ranks (or one)
    // both neighbours are the same peer, so the order matters: its first send (its highest slice, upwards) must
    // meet my first receive (into recv_lo), its second (its lowest slice, downwards) my second (into recv_hi).
    int rc = a->GroupStart();
    if (!rc) rc = a->Send(send_hi, bytes, kChar, up, t->comm, s);
    if (!rc) rc = a->Send(send_lo, bytes, kChar, dn, t->comm, s);
    if (!rc) rc = a->Recv(recv_lo, bytes, kChar, dn, t->comm, s);
    if (!rc) rc = a->Recv(recv_hi, bytes, kChar, up, t->comm, s);
    const int rc2 = a->GroupEnd();
    if (!rc) rc = rc2;
    t->last_error = rc;
    return rc ? -1 : 0;
}

inline int allreduce_sum(void* user, double* dev_buf, int n, void* stream) {
    Transport* t = (Transport*)user;
    Api* a = api(nullptr);
    if (!a || !t->comm) return -1;
    const int rc = a->AllReduce(dev_buf, dev_buf, (size_t)n, kFloat64, kSum, t->comm, (cudaStream_t)stream);
    t->last_error = rc;
    return rc ? -1 : 0;
}

}  // namespace lqcd_nccl

#endif
