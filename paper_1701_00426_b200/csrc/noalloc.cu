// noalloc.cu -- lqcd_mdagm_noalloc: the normal operator m^2 + sigma - D_eo D_oe (Eq. 8) for callers
// that have no device memory to give the library as workspace and are not allowed to obtain any.
//
// Who that is.  lqcd_mdagm needs one odd-site temporary (D_oe in_e) between its two Dslash launches and takes it
// from the workspace the caller handed to lqcd_set_workspace -- memory the caller had to get from somewhere.  Some
// callers cannot:
//   - a plug-in inside a host program that owns the whole device heap (a framework's caching allocator that has
//     already reserved the HBM, a job scheduler that gives each component a fixed arena and nothing more): a
//     cudaMalloc from inside the library would fail there, or take memory the owner believes it still has;
//   - a latency-critical loop (an HMC trajectory driven from a real-time or multi-tenant service): cudaMalloc and
//     cudaFree synchronise the whole device and may block behind other tenants' work, so they are banned after
//     start-up;
//   - a run sized to fill the GPU (links, solver vectors and the force fields of a large lattice planned to the
//     last GB of the 180 GB): there is no headroom left to ask for, and an allocation failure in the middle of
//     a trajectory would lose the run.
// For them the temporary lives in a file-scope `static __device__` array below.  It is part of the library's
// device image: the driver places it when the module is loaded onto a GPU, and every GPU that loads
// liblqcd_b200.so keeps those LQCD_NOALLOC_SCRATCH_BYTES bytes until the process exits, whether or not this entry
// point is ever called.  That is the price, and the reason the maximum is modest (8 MiB, i.e. up to 24^4 or
// 32^3 x 8 in fp64 and 32^3 x 16 in fp32); larger lattices are refused and must use lqcd_mdagm with a workspace.
//
// Host code cannot use the array's name as a pointer: on the host `g_noalloc_scratch` names a shadow object the
// compiler creates for registration, not device memory; a kernel handed &g_noalloc_scratch would fault, or --
// on a system where the GPU can reach pageable host memory -- quietly work on the wrong bytes.  The device
// address is asked for once per device with cudaGetSymbolAddress, with that device current, and that address is
// what the Dslash kernels receive as their `out` / `in` argument.
#include <mutex>

#include "common.cuh"

static __device__ __align__(256) unsigned char g_noalloc_scratch[LQCD_NOALLOC_SCRATCH_BYTES];

#define NOALLOC_MAX_DEVICES 64
static void *g_scratch_addr[NOALLOC_MAX_DEVICES];   // device address of g_noalloc_scratch on each ordinal (NULL: not asked yet)
static std::mutex g_scratch_mutex;

// The device address of the scratch array on ctx->device (which the caller has just made current).  The first
// call per device does the look-up; cudaGetSymbolAddress may make the runtime load this module onto the device,
// which is why that first call belongs to start-up, outside any stream capture.  No allocation is made here.
static int noalloc_scratch(lqcd_ctx *ctx, void **addr)
{
    const int dev = ctx->device;
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES)
        return lqcd_fail(ctx, LQCD_ERR_UNSUPPORTED, "lqcd_mdagm_noalloc: device ordinal %d >= %d", dev, NOALLOC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[dev]) {
        int cur = -1;
        cudaError_t e = cudaGetDevice(&cur);
        if (e != cudaSuccess) return lqcd_check_cuda(ctx, e, "lqcd_mdagm_noalloc: cudaGetDevice");
        if (cur != dev) return lqcd_fail(ctx, LQCD_ERR_CUDA, "lqcd_mdagm_noalloc: device %d is current, expected %d", cur, dev);
        void *p = NULL;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return lqcd_check_cuda(ctx, e, "lqcd_mdagm_noalloc: cudaGetSymbolAddress(static scratch)");
        if (!p || ((uintptr_t)p & 255))
            return lqcd_fail(ctx, LQCD_ERR_CUDA, "lqcd_mdagm_noalloc: static scratch at %p is not 256-byte aligned", p);
        g_scratch_addr[dev] = p;
    }
    *addr = g_scratch_addr[dev];
    return LQCD_OK;
}

extern "C" int lqcd_mdagm_noalloc(lqcd_ctx *ctx, void *out_e, const void *in_e, const void *links, double mass,
                                  double sigma)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (!out_e || !in_e || !links) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_mdagm_noalloc: null pointer");
    if (out_e == in_e) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_mdagm_noalloc: out and in alias");
    // slab contexts exchange halos between the two launches (hooks or the peer transport): not offered here, so
    // that the promise "no allocating call" does not depend on what a caller's hook does
    if (ctx->peer_on || ctx->peer_mem || ctx->halo_fn || ctx->x3_lo != 0 || ctx->x3_hi != ctx->g.N3)
        return lqcd_fail(ctx, LQCD_ERR_UNSUPPORTED, "lqcd_mdagm_noalloc: not available on a slab context");
    const size_t need = lqcd_spinor_bytes(ctx);
    if (need > (size_t)LQCD_NOALLOC_SCRATCH_BYTES)
        return lqcd_fail(ctx, LQCD_ERR_WORKSPACE,
                         "lqcd_mdagm_noalloc: one half-lattice vector of this context is %zu bytes, the static scratch holds "
                         "%zu; use lqcd_mdagm with a caller-owned workspace", need, (size_t)LQCD_NOALLOC_SCRATCH_BYTES);
    void *tmp_o = NULL;
    if ((rc = noalloc_scratch(ctx, &tmp_o))) return rc;
    // Nothing in the scratch has to start at zero: the first launch writes every element of the odd-site vector
    // (3 planes x Vh sites) and the second reads only those, so whatever the previous call left is overwritten
    // before it is read.  Stream order keeps the two launches of ONE call apart; two calls on different streams
    // (or from different contexts of this device) share the array and would race.
    const int par = ctx->solve_parity;     // LQCD_EVEN, as in lqcd_mdagm
    rc = launch_dslash(ctx, 1 - par, tmp_o, in_e, links, NULL, 0.0, 0, 0);
    if (rc) return rc;
    return launch_dslash(ctx, par, out_e, tmp_o, links, in_e, mass * mass + sigma, 0, 0);
}
