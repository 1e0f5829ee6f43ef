// peer.cuh -- device side of the slab mode's peer-to-peer transport ("direct P2P stores
// into the neighbour's ghost slice", two all-reduces of one double per CG iteration; the paper leaves the
// multi-device version as future work).
//
// Every rank owns one PeerBlock in its own device memory, mapped by all ranks of the node (cudaMalloc +
// CUDA IPC, or plain pointers when the ranks share a process).  Nothing here launches a kernel of its own in
// the CG loop except the face push: the PRODUCER of a partial sum publishes it to every rank's block from its
// last CTA, the CONSUMER kernel waits for the P flags at its start and adds the P slots in rank order (every
// rank gets the bit-identical total, so every rank takes the same decisions).  Halo: the push kernel stores the
// two boundary slices of a vector straight into the neighbours' landing buffers and raises their flag; the
// Dslash that reads the vector waits for its two flags and takes the x3 hops that leave the slab from the
// landing buffers (no unpack kernel, no ghost slices in the vectors are read).
//
// Flags carry monotone counters, never reset.  A rank's own counter of a sync point is, by construction, the
// value it must see from its peers: all ranks run the same sequence of sync points.  Re-use of a slot or a
// landing buffer is ordered by the all-reduces in between (solver.cu, "peer mode").
#pragma once
#include "common.cuh"

__device__ __forceinline__ unsigned int ld_flag(const unsigned int *p)
{
    unsigned int v;
    asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_flag(unsigned int *p, unsigned int v)
{
    asm volatile("st.release.sys.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void st_remote(double *p, double v)
{
    asm volatile("st.relaxed.sys.global.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}
__device__ __forceinline__ double ld_slot(const double *p)
{
    double v;
    asm volatile("ld.relaxed.sys.global.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}

// Called by ONE thread after the grid-wide local sum is complete (the last CTA of grid_sum_last, or a
// one-thread kernel): vals[0..nv) go to slot[kind][n & 1][rank][*] of every rank, then the flags.
__device__ __forceinline__ void peer_publish(const PeerDev &pd, int kind, const double *vals, int nv)
{
    const unsigned int n = pd.self->cnt_red[kind] + 1;
    pd.self->cnt_red[kind] = n;
    for (int r = 0; r < pd.nranks; ++r)
        for (int v = 0; v < nv; ++v) st_remote(&pd.peer[r]->slot[kind][n & 1][pd.rank][v], vals[v]);
    __threadfence_system();
    for (int r = 0; r < pd.nranks; ++r) st_flag(&pd.peer[r]->flag_red[kind][pd.rank], n);
}

// Called by every thread of a CTA at the start of the consumer kernel: wait until all ranks have published
// reduction number n = (own counter) of `kind`.  Ends with a CTA barrier.
__device__ __forceinline__ unsigned int peer_wait_red(const PeerDev &pd, int kind)
{
    const unsigned int n = *(volatile unsigned int *)&pd.self->cnt_red[kind];
    if (threadIdx.x < pd.nranks) {
        const unsigned int *f = &pd.self->flag_red[kind][threadIdx.x];
        while ((int)(ld_flag(f) - n) < 0) { }
    }
    __syncthreads();
    return n;
}
// sum over the ranks, in rank order, of value v of reduction n (after peer_wait_red)
__device__ __forceinline__ double peer_sum(const PeerDev &pd, int kind, unsigned int n, int v)
{
    double s = 0.0;
    for (int r = 0; r < pd.nranks; ++r) s += ld_slot(&pd.self->slot[kind][n & 1][r][v]);
    return s;
}

// Start of a Dslash that reads a vector whose faces were pushed as exchange `kind`: wait for both neighbours.
__device__ __forceinline__ void peer_wait_halo(const PeerDev &pd, int kind)
{
    const unsigned int n = *(volatile unsigned int *)&pd.self->cnt_halo[kind];
    if (threadIdx.x < 2) {
        const unsigned int *f = &pd.self->flag_halo[kind][threadIdx.x];
        while ((int)(ld_flag(f) - n) < 0) { }
    }
    __syncthreads();
}
