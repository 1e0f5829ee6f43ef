// peer.cuh -- device side of the slab mode's peer-to-peer transport ("direct P2P stores
// into the neighbour's ghost slice", two all-reduces of one double per CG iteration; the paper leaves the
// multi-device version as future work).
//
// Every rank owns one PeerBlock in its own device memory, mapped by all ranks of the node (cudaMalloc +
// CUDA IPC, or plain pointers when the ranks share a process).  Nothing here launches a kernel of its own in
// the CG loop except the face push, and no kernel of the loop uses a fence-and-ticket protocol: what orders a
// rank's own writes is the KERNEL BOUNDARY (every kernel starts with griddepcontrol.wait), what orders them for
// the peers is one release store per flag.
//   dot products: the producer (Dslash with <p,q>, K1 with <r,r>) leaves per-CTA partials as on a single GPU;
//     every CTA of the CONSUMER (K1, K2) adds them up for itself, CTA 0 stores the rank's sum into every rank's slot
//     and raises the flags; every CTA waits for the OTHER ranks' flags and adds the P sums in rank order (every rank
//     gets the bit-identical total, so every rank takes the same decisions);
//   halo: the push kernel stores the two boundary slices of a vector straight into the neighbours' landing
//     buffers; CTA 0 of the Dslash that follows it in the stream raises the neighbours' flags; only the tiles
//     of that Dslash that touch a boundary slice wait for the rank's own two flags, and they take the x3 hops
//     that leave the slab from the landing buffers (no unpack kernel; the vectors' ghost slices are not read).
//
// Flags carry monotone counters, never reset.  The counter of a sync point is bumped by one thread of the
// PRODUCING kernel (visible to the consumer through the kernel boundary); a rank's own counter is, by
// construction, the value it must see from its peers: all ranks run the same sequence of sync points.  Re-use of
// a slot or a landing buffer is ordered by the all-reduces in between (solver.cu, "peer mode").
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

// Spin until *f >= n (wrap-safe), but never for more than pd.wait_cycles (option peer_wait_ms, default 3 s): a peer that died or
// ran a different sequence of calls must not hang this GPU.  A wait that gives up counts itself in the rank's block, and
// from then on the transport of this rank is DEAD: every later wait (of this kernel's other CTAs, of every later kernel)
// returns at once instead of spending the limit again -- the flags are monotone counters, so a peer that missed one sync
// point misses all later ones, and 4 waits x 3 s per CG iteration would hold the GPU for hours.  The solver's host loop
// reads the count with every convergence poll and stops enqueueing (solver.cu); every call over a dead transport
// returns LQCD_ERR_CUDA (the results are meaningless) until lqcd_peer_disconnect + lqcd_peer_init build a new one.
__device__ __forceinline__ void peer_spin(const PeerDev &pd, const unsigned int *f, unsigned int n)
{
    if ((int)(ld_flag(f) - n) >= 0) return;
    if (*(volatile unsigned int *)&pd.self->timeouts) return;
    const long long t0 = clock64();
    while ((int)(ld_flag(f) - n) < 0) {
        if (clock64() - t0 > pd.wait_cycles) { atomicAdd(&pd.self->timeouts, 1u); return; }
        if (*(volatile unsigned int *)&pd.self->timeouts) return;      // another waiter of this rank gave up meanwhile
    }
}

// One thread of the producing kernel: this rank has one more reduction / exchange of `kind` under way.
__device__ __forceinline__ void peer_bump_red(const PeerDev &pd, int kind) { pd.self->cnt_red[kind] += 1; }
__device__ __forceinline__ void peer_bump_halo(const PeerDev &pd, int kind) { pd.self->cnt_halo[kind] += 1; }

// Called by ONE thread once the rank's local sum is complete: vals[0..nv) go to slot[kind][n & 1][rank][*] of
// every rank, then the flags (n = the rank's own counter of `kind`, bumped by the producing kernel).
__device__ __forceinline__ void peer_publish(const PeerDev &pd, int kind, const double *vals, int nv)
{
    const unsigned int n = *(volatile unsigned int *)&pd.self->cnt_red[kind];
    for (int r = 0; r < pd.nranks; ++r)
        for (int v = 0; v < nv; ++v) st_remote(&pd.peer[r]->slot[kind][n & 1][pd.rank][v], vals[v]);
    // (the release stores order the slots before the flags)
    for (int r = 0; r < pd.nranks; ++r) st_flag(&pd.peer[r]->flag_red[kind][pd.rank], n);
}

// Called by every thread of a CTA at the start of the consumer kernel: wait until all ranks have published
// reduction number n = (own counter) of `kind`.  Ends with a CTA barrier.
__device__ __forceinline__ unsigned int peer_wait_red(const PeerDev &pd, int kind)
{
    const unsigned int n = *(volatile unsigned int *)&pd.self->cnt_red[kind];
    if (threadIdx.x < pd.nranks) {
        peer_spin(pd, &pd.self->flag_red[kind][threadIdx.x], n);
    }
    __syncthreads();
    return n;
}
// The same for a consumer whose every CTA has already added up the rank's OWN partials (K1, K2: as on a single GPU, in
// parallel and bit-identically): only the OTHER ranks' flags are waited for, and `local` takes the rank's own place in
// the rank-ordered sum -- the rank never waits for its own publish / flag / poll round trip.
__device__ __forceinline__ double peer_gather_with_local(const PeerDev &pd, int kind, double local)
{
    const unsigned int n = *(volatile unsigned int *)&pd.self->cnt_red[kind];
    if (threadIdx.x < pd.nranks && threadIdx.x != pd.rank) peer_spin(pd, &pd.self->flag_red[kind][threadIdx.x], n);
    __syncthreads();
    double s = 0.0;
    for (int r = 0; r < pd.nranks; ++r) s += r == pd.rank ? local : ld_slot(&pd.self->slot[kind][n & 1][r][0]);
    return s;
}
// sum over the ranks, in rank order, of value v of reduction n (after peer_wait_red)
__device__ __forceinline__ double peer_sum(const PeerDev &pd, int kind, unsigned int n, int v)
{
    double s = 0.0;
    for (int r = 0; r < pd.nranks; ++r) s += ld_slot(&pd.self->slot[kind][n & 1][r][v]);
    return s;
}

// One thread of the Dslash that follows the push in the stream: the faces are in the neighbours' landing buffers
// (kernel boundary), tell them.
__device__ __forceinline__ void peer_signal_halo(const PeerDev &pd, int kind)
{
    const unsigned int n = *(volatile unsigned int *)&pd.self->cnt_halo[kind];
    st_flag(&pd.up->flag_halo[kind][0], n);        // the rank above sees its "from down" face
    st_flag(&pd.down->flag_halo[kind][1], n);
}
// A tile of that Dslash that reads a face: wait for both neighbours.
__device__ __forceinline__ void peer_wait_halo(const PeerDev &pd, int kind)
{
    const unsigned int n = *(volatile unsigned int *)&pd.self->cnt_halo[kind];
    if (threadIdx.x < 2) {
        peer_spin(pd, &pd.self->flag_halo[kind][threadIdx.x], n);
    }
    __syncthreads();
}
