// omni_slab.cuh -- z-slab sharding of one solve over several ranks.
//
// The paper stops at one 16 GB GPU and names memory as the limit.  The path shards along z: rank s
// owns the planes [z0_s, z1_s) and works on a WINDOW of the global grid, its planes plus up to two halo planes per
// side: two because the stencil codes of Eq. 25 (:266) read the validity of cells two planes away (the far cell of the
// F / B neighbour); one plane of every vector the operator is applied to is kept current by exchange.  The kernels are
// the single-device ones, restricted to the owned planes (Geom::kz0 / kz1); a window that touches the global box keeps
// the true face there, an artificial window end is never emitted.  Per CG iteration: one halo plane of p and one of r to
// each neighbour, two all-reduced scalars (gamma, rho'); per outer iteration: halo planes of delta, P and r and the
// four scalars of K2.  Every reduction leaves its per-rank total in Scalars::red_out (defer = 1), the totals are summed
// over the ranks, and a one-thread kernel runs the usual finalize code on every rank with identical numbers, so all
// ranks take the same decisions.
//
// Two transports behind one interface: all ranks in this process on this device (plane copies + a summing kernel:
// what one GPU can test), or one rank per process with NCCL over NVLink (ncclSend / ncclRecv + ncclAllReduce, the
// library loaded at run time).
#pragma once
#include <dlfcn.h>
#include "omni_kernels.cuh"

namespace omni {

// sum red_out[0..n) over the local ranks in rank order and give every rank the same totals
__global__ void slab_sum_kernel(Scalars* const* scs, int nranks, int n)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    for (int i = 0; i < n; ++i) {
        double t = 0.0;
        for (int s = 0; s < nranks; ++s) t += scs[s]->red_out[i];
        for (int s = 0; s < nranks; ++s) scs[s]->red_out[i] = t;
    }
}

__global__ void source_finalize_kernel(Scalars* sc) { source_finalize(sc, sc->red_out[0]); }

// ---- NCCL, loaded at run time (the library has no link-time dependency on it)
struct NcclApi {
    typedef struct { char internal[128]; } UniqueId;
    int (*GetUniqueId)(UniqueId*);
    int (*CommInitRank)(void**, int, UniqueId, int);
    int (*CommDestroy)(void*);
    int (*Send)(const void*, size_t, int, int, void*, cudaStream_t);
    int (*Recv)(void*, size_t, int, int, void*, cudaStream_t);
    int (*AllReduce)(const void*, void*, size_t, int, int, void*, cudaStream_t);
    int (*GroupStart)();
    int (*GroupEnd)();
    bool ok;
    enum { Int8 = 0, Float64 = 8, Sum = 0 };          // ncclDataType_t / ncclRedOp_t values of nccl.h
};

inline const NcclApi& nccl_api()
{
    static NcclApi api = {};
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* h = nullptr;
        const char* names[] = { "libnccl.so.2", "libnccl.so" };
        for (const char* n : names)
            if (!h) h = dlopen(n, RTLD_NOW | RTLD_GLOBAL);
        if (h) {
            api.GetUniqueId = (int (*)(NcclApi::UniqueId*))dlsym(h, "ncclGetUniqueId");
            api.CommInitRank = (int (*)(void**, int, NcclApi::UniqueId, int))dlsym(h, "ncclCommInitRank");
            api.CommDestroy = (int (*)(void*))dlsym(h, "ncclCommDestroy");
            api.Send = (int (*)(const void*, size_t, int, int, void*, cudaStream_t))dlsym(h, "ncclSend");
            api.Recv = (int (*)(void*, size_t, int, int, void*, cudaStream_t))dlsym(h, "ncclRecv");
            api.AllReduce = (int (*)(const void*, void*, size_t, int, int, void*, cudaStream_t))dlsym(h, "ncclAllReduce");
            api.GroupStart = (int (*)())dlsym(h, "ncclGroupStart");
            api.GroupEnd = (int (*)())dlsym(h, "ncclGroupEnd");
            api.ok = api.GetUniqueId && api.CommInitRank && api.CommDestroy && api.Send && api.Recv && api.AllReduce &&
                     api.GroupStart && api.GroupEnd;
        }
    }
    return api;
}

// owned planes [z0, z1) of rank `rank` (balanced: the first nz % nranks ranks own one plane more) and its window
// [zlo, zhi) = owned planes plus up to two halo planes per side
inline bool slab_plan(int nz, int nranks, int rank, int& z0, int& z1, int& zlo, int& zhi)
{
    if (nranks < 1 || rank < 0 || rank >= nranks || nz < nranks) return false;
    const int q = nz / nranks, rem = nz % nranks;
    z0 = rank * q + (rank < rem ? rank : rem);
    z1 = z0 + q + (rank < rem ? 1 : 0);
    zlo = z0 - 2 < 0 ? 0 : z0 - 2;
    zhi = z1 + 2 > nz ? nz : z1 + 2;
    return true;
}

}  // namespace omni
