// pack.cu -- canonical (AoS, lexicographic, complex128) <-> native (parity-split SoA) fields.
// Step a1 of SURVEY.md section 8(a): PAPER.md:245-272 (SoA vec3_soa / su3_soa, Figs 1-2), the even-site
// index of Eq. 9, and the 2-row link storage of PAPER.md:272 (row 2 dropped
// here, rebuilt in registers by the Dslash kernel).  Setup cost, untimed.
#include "common.cuh"

// idxh, parity -> lexicographic site index
__device__ __forceinline__ int lex_of_half(const Geom &g, int i, int parity)
{
    uint32_t t = fd_div((uint32_t)i, g.dNh0);
    uint32_t t2 = fd_div(t, g.dN1);
    int x1 = (int)t - (int)t2 * g.N1;
    uint32_t x3 = fd_div(t2, g.dN2);
    int x2 = (int)t2 - (int)x3 * g.N2;
    int rp = (x1 + x2 + (int)x3 + parity) & 1;
    return 2 * i + rp;     // lex = 2*idxh + (x0 & 1), and x0 = 2*hx0 + rp
}

template <typename T, int LAYOUT>
__global__ void pack_links_kernel(Geom g, int rows, T *__restrict__ native, const double2 *__restrict__ canon)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int par = blockIdx.y;
    if (i >= g.Vh) return;
    size_t lex = (size_t)lex_of_half(g, i, par);
    for (int mu = 0; mu < 4; ++mu)
        for (int r = 0; r < rows; ++r)
            for (int c = 0; c < 3; ++c) {
                double2 z = canon[(lex * 4 + mu) * 9 + r * 3 + c];
                size_t plane = ((size_t)(par * 4 + mu) * rows + r) * 3 + c;
                st_cx<T, LAYOUT, 0>(native, plane, (size_t)g.Ls, (size_t)i, cx<T>((T)z.x, (T)z.y), L2Pol());
            }
}

// backfield theta[lex][mu] (one real per link, the paper's double_soa argument of acc_Deo)
// -> native [parity][mu][idxh]
// format 0: theta itself; format 1: (cos theta, sin theta), evaluated here in fp64 and rounded once
template <typename T>
__global__ void pack_backfield_kernel(Geom g, int format, T *__restrict__ native, const double *__restrict__ canon)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int par = blockIdx.y;
    if (i >= g.Vh) return;
    size_t lex = (size_t)lex_of_half(g, i, par);
    for (int mu = 0; mu < 4; ++mu) {
        const double th = canon[lex * 4 + mu];
        const size_t k = (size_t)(par * 4 + mu) * g.Vh + i;
        if (format == 0) native[k] = (T)th;
        else { double sn, cs; sincos(th, &sn, &cs); native[2 * k] = (T)cs; native[2 * k + 1] = (T)sn; }
    }
}

template <typename T, int LAYOUT>
__global__ void pack_spinor_kernel(Geom g, T *__restrict__ native, const double2 *__restrict__ canon)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.Vh) return;
    for (int c = 0; c < 3; ++c) {
        double2 z = canon[(size_t)i * 3 + c];
        st_cx<T, LAYOUT, 0>(native, (size_t)c, (size_t)g.Vh, (size_t)i, cx<T>((T)z.x, (T)z.y), L2Pol());
    }
}

template <typename T, int LAYOUT>
__global__ void unpack_spinor_kernel(Geom g, double2 *__restrict__ canon, const T *__restrict__ native)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.Vh) return;
    for (int c = 0; c < 3; ++c) {
        Cx<T> z = ld_cx<T, LAYOUT, 0, 0>(native, (size_t)c, (size_t)g.Vh, (size_t)i, L2Pol());
        canon[(size_t)i * 3 + c] = make_double2((double)z.re, (double)z.im);
    }
}

// One x3 slice (s3 = Nh0*N1*N2 sites) of a native half vector <-> a contiguous buffer laid out like a
// half vector of s3 sites.  PACK: buf = sign * slice; else slice = buf.  (Slab mode halo, lqcd.h.)
// blockIdx.y selects one of up to two faces handled by the same launch (buf / x3 / sign of face 0 or 1).
template <typename T, int LAYOUT, int PACK>
__global__ void halo_kernel(Geom g, T *__restrict__ buf0, T *__restrict__ buf1, T *__restrict__ spinor, int x3_0, int x3_1,
                            T sign0, T sign1)
{
    pdl_wait();
    pdl_trigger();
    T *__restrict__ buf = blockIdx.y ? buf1 : buf0;
    const int x3 = blockIdx.y ? x3_1 : x3_0;
    const T sign = blockIdx.y ? sign1 : sign0;
    int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= g.s3) return;
    const size_t i = (size_t)x3 * g.s3 + f;
    for (int c = 0; c < 3; ++c) {
        if (PACK) {
            Cx<T> z = ld_cx<T, LAYOUT, 0, 0>(spinor, (size_t)c, (size_t)g.Vh, i, L2Pol());
            st_cx<T, LAYOUT, 0>(buf, (size_t)c, (size_t)g.s3, (size_t)f, cx<T>(sign * z.re, sign * z.im), L2Pol());
        } else {
            // plain (coherent) load: the buffer was just written by a copy / another rank
            Cx<T> z;
            if (LAYOUT == 0) {
                typedef typename Vec2<T>::type V2;
                V2 v = reinterpret_cast<const V2 *>(buf)[(size_t)c * g.s3 + f];
                z = cx<T>(v.x, v.y);
            } else {
                z = cx<T>(buf[(size_t)(2 * c) * g.s3 + f], buf[(size_t)(2 * c + 1) * g.s3 + f]);
            }
            st_cx<T, LAYOUT, 0>(spinor, (size_t)c, (size_t)g.Vh, i, z, L2Pol());
        }
    }
}

#define DISPATCH_TL(ctx, CALL)                                             \
    do {                                                                   \
        if ((ctx)->prec == LQCD_F64) {                                     \
            if ((ctx)->layout == 0) { CALL(double, 0); } else { CALL(double, 1); } \
        } else {                                                           \
            if ((ctx)->layout == 0) { CALL(float, 0); } else { CALL(float, 1); }   \
        }                                                                  \
    } while (0)

int launch_pack_links(lqcd_ctx *ctx, void *native, const void *canonical)
{
    int rows = ctx->recon == LQCD_RECON_12 ? 2 : 3;
    dim3 grid((ctx->g.Vh + 127) / 128, 2), block(128);
#define CALL(T, L) pack_links_kernel<T, L><<<grid, block, 0, ctx->stream>>>(ctx->g, rows, (T *)native, (const double2 *)canonical)
    DISPATCH_TL(ctx, CALL);
#undef CALL
    ctx->launches++;
    return lqcd_check_cuda(ctx, cudaGetLastError(), "pack_links");
}

int launch_pack_backfield(lqcd_ctx *ctx, void *native, const void *canonical)
{
    dim3 grid((ctx->g.Vh + 127) / 128, 2), block(128);
    if (ctx->prec == LQCD_F64) pack_backfield_kernel<double><<<grid, block, 0, ctx->stream>>>(ctx->g, ctx->backfield_format, (double *)native, (const double *)canonical);
    else pack_backfield_kernel<float><<<grid, block, 0, ctx->stream>>>(ctx->g, ctx->backfield_format, (float *)native, (const double *)canonical);
    ctx->launches++;
    return lqcd_check_cuda(ctx, cudaGetLastError(), "pack_backfield");
}

int launch_pack_spinor(lqcd_ctx *ctx, int parity, void *native, const void *canonical)
{
    (void)parity;  // the half-lattice order idxh = lex/2 is the same for both parities (Eq. 9)
    dim3 grid((ctx->g.Vh + 127) / 128), block(128);
#define CALL(T, L) pack_spinor_kernel<T, L><<<grid, block, 0, ctx->stream>>>(ctx->g, (T *)native, (const double2 *)canonical)
    DISPATCH_TL(ctx, CALL);
#undef CALL
    ctx->launches++;
    return lqcd_check_cuda(ctx, cudaGetLastError(), "pack_spinor");
}

int launch_unpack_spinor(lqcd_ctx *ctx, int parity, void *canonical, const void *native)
{
    (void)parity;
    dim3 grid((ctx->g.Vh + 127) / 128), block(128);
#define CALL(T, L) unpack_spinor_kernel<T, L><<<grid, block, 0, ctx->stream>>>(ctx->g, (double2 *)canonical, (const T *)native)
    DISPATCH_TL(ctx, CALL);
#undef CALL
    ctx->launches++;
    return lqcd_check_cuda(ctx, cudaGetLastError(), "unpack_spinor");
}

int launch_halo(lqcd_ctx *ctx, int pack, void *buf, void *spinor, int x3, double sign)
{
    return launch_halo2(ctx, pack, buf, NULL, spinor, x3, 0, sign, 1.0);
}

// one launch for both faces (buf1 == NULL: one face only)
int launch_halo2(lqcd_ctx *ctx, int pack, void *buf0, void *buf1, void *spinor, int x3_0, int x3_1, double sign0, double sign1)
{
    dim3 grid((ctx->g.s3 + 127) / 128, buf1 ? 2 : 1), block(128);
#define CALL(T, L) do { if (pack) launch_k(ctx, halo_kernel<T, L, 1>, grid, block, ctx->g, (T *)buf0, (T *)buf1, (T *)spinor, x3_0, x3_1, (T)sign0, (T)sign1); \
                        else launch_k(ctx, halo_kernel<T, L, 0>, grid, block, ctx->g, (T *)buf0, (T *)buf1, (T *)spinor, x3_0, x3_1, (T)sign0, (T)sign1); } while (0)
    DISPATCH_TL(ctx, CALL);
#undef CALL
    return lqcd_check_cuda(ctx, cudaGetLastError(), "halo");
}
