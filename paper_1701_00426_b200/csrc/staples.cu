// staples.cu -- gauge staples of the tree-level Symanzik improved action.
// PAPER.md:105 names the action; "the computation of staples in the gauge force calculation
// is the most time consuming [task of the gauge cycles].  It consists of calculating 6 products of 3 and
// 5 SU(3) matrices representing links on C-shaped paths"; Listing 3 shows only the
// loop nest, with indirect neighbour addressing.  Paths and coefficients: reading R22 of DESIGN.md:
//
//   W[U] = sum_x sum_{mu<nu} { c0 Re Tr P_{mu nu}(x) + c1 [Re Tr R_{mu nu}(x) + Re Tr R_{nu mu}(x)] },
//   c0 = 5/3, c1 = -1/12;   S_mu(x) = sum over the loops of W through U_mu(x) of coefficient x (the
//   remaining links ordered from x+mu back to x):  W = Re Tr[U_mu(x) S_mu(x)] + (terms without U_mu(x)).
//
// Per nu != mu: 2 three-link paths (plaquette) and 6 five-link paths (2x1 rectangles).  A path is walked
// from x+mu: a step +d from y multiplies by U_d(y), a step -d by U_d(y-d)^dagger.  Periodic links.
//
// One thread per link (x, mu): CTA = 128 consecutive sites of one parity, blockIdx.y = mu, blockIdx.z =
// parity.  Unlike the paper's kernel there are no neighbour tables: the walker keeps the coordinates in
// registers and computes (parity, idxh) of every visited site arithmetically.  84 3x3 complex products and
// 108 link loads per output link: the kernel is bound by FP64 FMA issue and L1/L2 bandwidth, not by HBM
// (algorithmic HBM traffic is 576 B in + 576 B out per site, ~0.2 ns/site at the measured peak).
#include "su3.cuh"

// step codes: bit 1 = direction (0: mu, 1: nu), bit 0 = sign (0: +, 1: -); 0xF terminates 3-link paths
#define SM_P 0
#define SM_M 1
#define SN_P 2
#define SN_M 3
__constant__ unsigned char c_paths[8][5] = {
    { SN_P, SM_M, SN_M, 0xF, 0xF },           // plaquette, above
    { SN_M, SM_M, SN_P, 0xF, 0xF },           // plaquette, below
    { SM_P, SN_P, SM_M, SM_M, SN_M },         // 2x1 along mu, link = first long side, above
    { SM_P, SN_M, SM_M, SM_M, SN_P },         //                                       below
    { SN_P, SM_M, SM_M, SN_M, SM_P },         // 2x1 along mu, link = second long side, above
    { SN_M, SM_M, SM_M, SN_P, SM_P },         //                                        below
    { SN_P, SN_P, SM_M, SN_M, SN_M },         // 1x2 along nu, link = short side, above
    { SN_M, SN_M, SM_M, SN_P, SN_P },         //                                  below
};

template <typename T> __device__ __forceinline__ void mat_mul_nn(Su3<T> &m, const Su3<T> &l)      // m = m l
{
    Su3<T> o;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            T re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                re = fma(m.e[a][k].re, l.e[k][b].re, re);
                re = fma(-m.e[a][k].im, l.e[k][b].im, re);
                im = fma(m.e[a][k].re, l.e[k][b].im, im);
                im = fma(m.e[a][k].im, l.e[k][b].re, im);
            }
            o.e[a][b] = cx<T>(re, im);
        }
    m = o;
}
template <typename T> __device__ __forceinline__ void mat_mul_nd(Su3<T> &m, const Su3<T> &l)      // m = m l^dagger
{
    Su3<T> o;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            T re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                re = fma(m.e[a][k].re, l.e[b][k].re, re);
                re = fma(m.e[a][k].im, l.e[b][k].im, re);
                im = fma(m.e[a][k].im, l.e[b][k].re, im);
                im = fma(-m.e[a][k].re, l.e[b][k].im, im);
            }
            o.e[a][b] = cx<T>(re, im);
        }
    m = o;
}

struct Site4 { int x0, x1, x2, x3; };
__device__ __forceinline__ void site_step(Site4 &s, const Geom &g, int d, int neg)
{
    // coordinates stay in registers: no dynamically indexed array
    if (d == 0) s.x0 = neg ? (s.x0 == 0 ? g.N0 - 1 : s.x0 - 1) : (s.x0 + 1 == g.N0 ? 0 : s.x0 + 1);
    else if (d == 1) s.x1 = neg ? (s.x1 == 0 ? g.N1 - 1 : s.x1 - 1) : (s.x1 + 1 == g.N1 ? 0 : s.x1 + 1);
    else if (d == 2) s.x2 = neg ? (s.x2 == 0 ? g.N2 - 1 : s.x2 - 1) : (s.x2 + 1 == g.N2 ? 0 : s.x2 + 1);
    else s.x3 = neg ? (s.x3 == 0 ? g.N3 - 1 : s.x3 - 1) : (s.x3 + 1 == g.N3 ? 0 : s.x3 + 1);
}

// CTA -> (site tile, mu, parity).  A link is needed again by staples two x3 slices away; in plain idxh
// order that reuse distance is 4-5 full time slices of links (94 MB at 32^4: ncu showed 8.6 GB of DRAM
// reads per launch against 0.6 GB of links).  The swizzle (a) makes (mu, parity) the fastest index, so
// that the 8 CTAs of one site tile run together, and (b) sweeps x3 inside blocks of `x2b` values of x2,
// which cuts the x3 reuse distance to x2b/N2 of a slice.  tiles_row = tiles of 128 sites per (x2, x3)
// row; sw.x2b == 0: identity order.
struct StapleSwizzle { int x2b, tiles_row, N2, N3; };
__device__ __forceinline__ void staple_cta(const StapleSwizzle &sw, int &tile, int &mu, int &parity)
{
    const int bid = blockIdx.x;
    parity = bid & 1;
    mu = (bid >> 1) & 3;
    int t = bid >> 3;
    if (sw.x2b > 0) {
        // t enumerates (b, x3, j, tx) with x2 = b*x2b + j, tx the tile inside the row
        const int tx = t % sw.tiles_row; t /= sw.tiles_row;
        const int j = t % sw.x2b; t /= sw.x2b;
        const int x3 = t % sw.N3;
        const int b = t / sw.N3;
        t = tx + sw.tiles_row * ((b * sw.x2b + j) + sw.N2 * x3);
    }
    tile = t;
}

template <typename T, int LAYOUT, int RECON12>
__global__ void __launch_bounds__(128, 3) staples_kernel(const Geom g, T *__restrict__ staples, const T *__restrict__ links,
                                                      const T c0, const T c1, const StapleSwizzle sw)
{
    pdl_wait();
    pdl_trigger();
    int tile, mu, parity;
    staple_cta(sw, tile, mu, parity);
    const int i = tile * blockDim.x + threadIdx.x;
    if (i >= g.Vh) return;
    const L2Pol pol = {0, 0};
    uint32_t t = fd_div((uint32_t)i, g.dNh0);
    const int hx0 = i - (int)t * g.Nh0;
    uint32_t t2 = fd_div(t, g.dN1);
    Site4 x;
    x.x1 = (int)t - (int)t2 * g.N1;
    x.x3 = (int)fd_div(t2, g.dN2);
    x.x2 = (int)t2 - x.x3 * g.N2;
    x.x0 = 2 * hx0 + ((x.x1 + x.x2 + x.x3 + parity) & 1);
    Site4 xm = x;
    site_step(xm, g, mu, 0);                       // every path starts at x + mu

    Su3<T> S;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) S.e[a][b] = cx<T>((T)0, (T)0);

    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
#pragma unroll 1
        for (int p = 0; p < 8; ++p) {
            // Addresses depend only on the path, not on the running product: resolve all steps first so
            // that the link loads of a path are issued back to back, ahead of the dependent products.
            const int nsteps = p < 2 ? 3 : 5;
            Site4 y = xm;
            int spar[5], sdir[5], sneg[5];
            size_t sidx[5];
#pragma unroll
            for (int s = 0; s < 5; ++s) {
                const int code = c_paths[p][s < nsteps ? s : 0];
                const int d = (code & 2) ? nu : mu, neg = code & 1;
                if (neg) site_step(y, g, d, 1);    // U_d(y-d)^dagger lives at y-d
                spar[s] = (y.x0 + y.x1 + y.x2 + y.x3) & 1;
                sidx[s] = (size_t)((y.x0 >> 1) + g.Nh0 * (y.x1 + g.N1 * (y.x2 + g.N2 * y.x3)));
                sdir[s] = d; sneg[s] = neg;
                if (!neg) site_step(y, g, d, 0);
            }
            Su3<T> M = load_link<T, LAYOUT, RECON12, 0, 0>(links, spar[0], sdir[0], (size_t)g.Ls, sidx[0], pol);
            if (sneg[0]) {
                Su3<T> D;
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) D.e[a][b] = cx<T>(M.e[b][a].re, -M.e[b][a].im);
                M = D;
            }
#pragma unroll
            for (int s = 1; s < 5; ++s) {
                if (s < nsteps) {
                    const Su3<T> L = load_link<T, LAYOUT, RECON12, 0, 0>(links, spar[s], sdir[s], (size_t)g.Ls, sidx[s], pol);
                    if (sneg[s]) mat_mul_nd<T>(M, L); else mat_mul_nn<T>(M, L);
                }
            }
            const T c = p < 2 ? c0 : c1;
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    S.e[a][b].re = fma(c, M.e[a][b].re, S.e[a][b].re);
                    S.e[a][b].im = fma(c, M.e[a][b].im, S.e[a][b].im);
                }
        }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b)
            st_cx<T, LAYOUT, 0>(staples, (size_t)((parity * 4 + mu) * 9 + a * 3 + b), (size_t)g.Vh, (size_t)i, S.e[a][b], pol);
}

// ---------------------------------------------------------------------------------------------
// Variant 1 (option staples_variant = 1): the eight paths of one (mu, nu) share sub-products.
// With m = mu^, n = nu^ and, above the link,
//   A = U_nu(x+m), B = U_mu(x+n)^+, C = U_nu(x)^+,
//   X = U_mu(x+m) U_nu(x+2m) U_mu(x+m+n)^+,  Y = U_mu(x-m+n)^+ U_nu(x-m)^+ U_mu(x-m),
//   Z = U_nu(x+m+n) U_mu(x+2n)^+ U_nu(x+n)^+ :
//   c0 ABC + c1 (XBC + ABY + AZC) = (c0 A + c1 X)(BC) + c1 A (BY + ZC)
// and the mirror image below the link: 22 products and 28 link loads per nu instead of 28 and 36.
// ---------------------------------------------------------------------------------------------
template <typename T> __device__ __forceinline__ Su3<T> mm(const Su3<T> &a, const Su3<T> &b)
{
    Su3<T> o = a;
    mat_mul_nn<T>(o, b);
    return o;
}
template <typename T> __device__ __forceinline__ Su3<T> dagger(const Su3<T> &l)
{
    Su3<T> d;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) d.e[a][b] = cx<T>(l.e[b][a].re, -l.e[b][a].im);
    return d;
}
// lin = ca a + cb b
template <typename T> __device__ __forceinline__ Su3<T> lin(T ca, const Su3<T> &a, T cb, const Su3<T> &b)
{
    Su3<T> o;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j)
            o.e[i][j] = cx<T>(fma(ca, a.e[i][j].re, cb * b.e[i][j].re), fma(ca, a.e[i][j].im, cb * b.e[i][j].im));
    return o;
}
__device__ __forceinline__ int wrap_coord(int c, int N) { return c >= N ? c - N : (c < 0 ? c + N : c); }
__device__ __forceinline__ int coord_of(const Site4 &s, int d) { return d == 0 ? s.x0 : d == 1 ? s.x1 : d == 2 ? s.x2 : s.x3; }
__device__ __forceinline__ int extent_of(const Geom &g, int d) { return d == 0 ? g.N0 : d == 1 ? g.N1 : d == 2 ? g.N2 : g.N3; }
__device__ __forceinline__ void set_coord(Site4 &s, int d, int v)
{
    if (d == 0) s.x0 = v; else if (d == 1) s.x1 = v; else if (d == 2) s.x2 = v; else s.x3 = v;
}

// U_dir(x + dm m + dn n), optionally daggered
template <typename T, int LAYOUT, int RECON12>
__device__ __forceinline__ Su3<T> link_at(const T *__restrict__ links, const Geom &g, const Site4 &x, int mu, int dm,
                                          int nu, int dn, int dir, bool dag)
{
    Site4 y = x;
    set_coord(y, mu, wrap_coord(coord_of(x, mu) + dm, extent_of(g, mu)));
    set_coord(y, nu, wrap_coord(coord_of(x, nu) + dn, extent_of(g, nu)));
    const int par = (y.x0 + y.x1 + y.x2 + y.x3) & 1;
    const size_t idx = (size_t)((y.x0 >> 1) + g.Nh0 * (y.x1 + g.N1 * (y.x2 + g.N2 * y.x3)));
    const L2Pol pol = {0, 0};
    const Su3<T> L = load_link<T, LAYOUT, RECON12, 0, 0>(links, par, dir, (size_t)g.Ls, idx, pol);
    return dag ? dagger<T>(L) : L;
}

// idxh displacement of the site x + k d^ relative to x (periodic wrap included).  Direction 0 moves the
// half-index by (x0' >> 1) - (x0 >> 1); the others by whole strides.  The parity of the displaced site is
// parity ^ (k & 1) (all extents are even).  With these per-thread tables a link address is
// i + dmu[dm] + dnu[dn]: two adds instead of a coordinate walk per load.
__device__ __forceinline__ int idxh_disp(const Geom &g, const Site4 &x, int d, int k)
{
    const int c = coord_of(x, d), N = extent_of(g, d);
    const int c2 = wrap_coord(c + k, N);
    if (d == 0) return (c2 >> 1) - (c >> 1);
    const int stride = d == 1 ? g.s1 : d == 2 ? g.s2 : g.s3;
    return (c2 - c) * stride;
}

template <typename T, int LAYOUT, int RECON12>
__device__ __forceinline__ Su3<T> link_rel(const T *__restrict__ links, const Geom &g, int i, int par, int disp, int dir, bool dag)
{
    const L2Pol pol = {0, 0};
    const Su3<T> L = load_link<T, LAYOUT, RECON12, 0, 0>(links, par, dir, (size_t)g.Ls, (size_t)(i + disp), pol);
    return dag ? dagger<T>(L) : L;
}

template <typename T, int LAYOUT>
__device__ __forceinline__ void store_mat_stream(T *__restrict__ f, size_t plane0, size_t Vh, size_t i, const Su3<T> &m);

template <typename T, int LAYOUT, int RECON12>
__global__ void __launch_bounds__(128, 2) staples_kernel_shared(const Geom g, T *__restrict__ staples,
                                                                const T *__restrict__ links, const T c0, const T c1, const StapleSwizzle sw)
{
    pdl_wait();
    pdl_trigger();
    int tile, mu, parity;
    staple_cta(sw, tile, mu, parity);
    const int i = tile * blockDim.x + threadIdx.x;
    if (i >= g.Vh) return;
    uint32_t t = fd_div((uint32_t)i, g.dNh0);
    const int hx0 = i - (int)t * g.Nh0;
    uint32_t t2 = fd_div(t, g.dN1);
    Site4 x;
    x.x1 = (int)t - (int)t2 * g.N1;
    x.x3 = (int)fd_div(t2, g.dN2);
    x.x2 = (int)t2 - x.x3 * g.N2;
    x.x0 = 2 * hx0 + ((x.x1 + x.x2 + x.x3 + parity) & 1);
    // base pointers of the four link blocks this thread reads: (own / other parity) x (mu / nu)
    constexpr int R3 = (RECON12 ? 2 : 3) * 3;
    const T *const bm0 = links + 2 * (size_t)((parity * 4 + mu) * R3) * g.Ls;
    const T *const bm1 = links + 2 * (size_t)(((parity ^ 1) * 4 + mu) * R3) * g.Ls;
#define LKM(dm, dn, dag) link_rel<T, LAYOUT, RECON12>((((dm) + (dn)) & 1) ? bm1 : bm0, g, i, 0, dmu[(dm) + 1] + dnu[(dn) + 2], 0, dag)
#define LKN(dm, dn, dag) link_rel<T, LAYOUT, RECON12>((((dm) + (dn)) & 1) ? bn1 : bn0, g, i, 0, dmu[(dm) + 1] + dnu[(dn) + 2], 0, dag)
    Su3<T> S;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) S.e[a][b] = cx<T>((T)0, (T)0);
    int dmu[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) dmu[k] = idxh_disp(g, x, mu, k - 1);
#pragma unroll 1
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        int dnu[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) dnu[k] = idxh_disp(g, x, nu, k - 2);
        const T *const bn0 = links + 2 * (size_t)((parity * 4 + nu) * R3) * g.Ls;
        const T *const bn1 = links + 2 * (size_t)(((parity ^ 1) * 4 + nu) * R3) * g.Ls;
        // Order chosen for short live ranges (an fp64 SU(3) matrix is 36 registers): W = BY + ZC first,
        // then A W, then (c0 A + c1 X)(BC); B and C are re-read from L1 rather than kept.
        {   // above the link
            Su3<T> W = mm<T>(LKM(0, 1, true),
                             mm<T>(mm<T>(LKM(-1, 1, true), LKN(-1, 0, true)), LKM(-1, 0, false)));      // B Y
            {
                const Su3<T> ZC = mm<T>(mm<T>(mm<T>(LKN(1, 1, false), LKM(0, 2, true)), LKN(0, 1, true)),
                                        LKN(0, 0, true));                                                  // Z C
                W = lin<T>((T)1, W, (T)1, ZC);
            }
            const Su3<T> A = LKN(1, 0, false);
            S = lin<T>((T)1, S, c1, mm<T>(A, W));
            const Su3<T> X = lin<T>(c0, A, c1, mm<T>(mm<T>(LKM(1, 0, false), LKN(2, 0, false)), LKM(1, 1, true)));
            const Su3<T> BC = mm<T>(LKM(0, 1, true), LKN(0, 0, true));
            S = lin<T>((T)1, S, (T)1, mm<T>(X, BC));
        }
        {   // below the link
            Su3<T> W = mm<T>(LKM(0, -1, true),
                             mm<T>(mm<T>(LKM(-1, -1, true), LKN(-1, -1, false)), LKM(-1, 0, false)));    // B' Y'
            {
                const Su3<T> ZC = mm<T>(mm<T>(mm<T>(LKN(1, -2, true), LKM(0, -2, true)), LKN(0, -2, false)),
                                        LKN(0, -1, false));                                                // Z' C'
                W = lin<T>((T)1, W, (T)1, ZC);
            }
            const Su3<T> A = LKN(1, -1, true);
            S = lin<T>((T)1, S, c1, mm<T>(A, W));
            const Su3<T> X = lin<T>(c0, A, c1, mm<T>(mm<T>(LKM(1, 0, false), LKN(2, -1, true)), LKM(1, -1, true)));
            const Su3<T> BC = mm<T>(LKM(0, -1, true), LKN(0, -1, false));
            S = lin<T>((T)1, S, (T)1, mm<T>(X, BC));
        }
    }
#undef LKM
#undef LKN
    // streaming stores: the output must not evict the link neighbourhood from L2 (round 1: 855 MB written to DRAM
    // against 604 MB of output)
    store_mat_stream<T, LAYOUT>(staples, (size_t)((parity * 4 + mu) * 9), (size_t)g.Vh, (size_t)i, S);
}


// ---------------------------------------------------------------------------------------------
// Variant 2 (option staples_variant = 2, the default when the workspace is large enough): two passes
// through 24 intermediate fields per site, the 3-link staples of every ordered pair (m, n), m != n,
//   Tu_mn(x) = U_n(x+m) U_m(x+n)^+ U_n(x)^+          (above the link U_m(x); the plaquette staple itself)
//   Tl_mn(x) = U_n(x+m-n)^+ U_m(x-n)^+ U_n(x-n)       (below)
// Every 5-link rectangle path through U_mu(x) is a 3-link staple of a NEIGHBOURING link times two links
// (no unitarity is used: these are regroupings of the same ordered products):
//   above:  U_mu(x+mu) U_nu(x+2mu) U_mu(x+mu+nu)^+ . B C  = Tu_numu(x+mu)^+ B C        B = U_mu(x+nu)^+
//           A B . U_mu(x-mu+nu)^+ U_nu(x-mu)^+ U_mu(x-mu) = A B Tl_numu(x)             A = U_nu(x+mu)
//           A . U_nu(x+mu+nu) U_mu(x+2nu)^+ U_nu(x+nu)^+ . C = A Tu_munu(x+nu) C      C = U_nu(x)^+
//   below:  Tu_numu(x+mu-nu) B' C',  A' B' Tl_numu(x-nu)^+,  A' Tl_munu(x-nu) C'
//           A' = U_nu(x+mu-nu)^+, B' = U_mu(x-nu)^+, C' = U_nu(x-nu)
//   S_mu(x) = sum_nu  c0 [Tu_munu(x) + Tl_munu(x)]
//                   + c1 { [Tu_numu(x+mu)^+ B + A Tu_munu(x+nu)] C + (A B) Tl_numu(x) }
//                   + c1 { [Tu_numu(x+mu-nu) B' + A' Tl_munu(x-nu)] C' + (A' B') Tl_numu(x-nu)^+ }
// Pass 1 (staples_produce_kernel, one thread per site and ordered pair): Q = U_m(y) U_n(y+m), then
//   Tl_mn(y+n) = Q^+ U_n(y) and Tu_nm(y) = U_m(y+n) Q^+ : 3 products for 2 fields, 36 per site.
// Pass 2 (staples_final_kernel, one thread per link): 10 products and 14 matrix loads per nu.
// 39 products per link instead of 66 (variant 1) / 84 (the definition); the price is 24 x 144 B per site of
// intermediate fields written and read once (fp64): the work moves from the FP64 pipe to HBM.
// ---------------------------------------------------------------------------------------------
__host__ __device__ __forceinline__ int pair_idx(int m, int n) { return m * 3 + (n < m ? n : n - 1); }
// first plane of the field of `kind` (0: Tu, 1: Tl) of the ordered pair q on the sites of parity par
__device__ __forceinline__ size_t tfield_plane(int par, int q, int kind) { return (size_t)(((par * 12 + q) * 2 + kind) * 9); }

// op(a) op(b), op = dagger when the flag is set
template <typename T, int DA, int DB> __device__ __forceinline__ Su3<T> mul_op(const Su3<T> &a, const Su3<T> &b)
{
    Su3<T> o;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = 0, im = 0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const T ar = DA ? a.e[k][i].re : a.e[i][k].re, ai = DA ? -a.e[k][i].im : a.e[i][k].im;
                const T br = DB ? b.e[j][k].re : b.e[k][j].re, bi = DB ? -b.e[j][k].im : b.e[k][j].im;
                re = fma(ar, br, re);
                re = fma(-ai, bi, re);
                im = fma(ar, bi, im);
                im = fma(ai, br, im);
            }
            o.e[i][j] = cx<T>(re, im);
        }
    return o;
}
// s += c * op(m)
template <typename T, int DM> __device__ __forceinline__ void acc_op(Su3<T> &s, T c, const Su3<T> &m)
{
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            s.e[i][j].re = fma(c, DM ? m.e[j][i].re : m.e[i][j].re, s.e[i][j].re);
            s.e[i][j].im = fma(DM ? -c : c, DM ? m.e[j][i].im : m.e[i][j].im, s.e[i][j].im);
        }
}
// x = cx * x + cm * op(m)
template <typename T, int DM> __device__ __forceinline__ void scale_acc_op(Su3<T> &x, T cx_, T cm, const Su3<T> &m)
{
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            x.e[i][j].re = fma(cx_, x.e[i][j].re, cm * (DM ? m.e[j][i].re : m.e[i][j].re));
            x.e[i][j].im = fma(cx_, x.e[i][j].im, (DM ? -cm : cm) * (DM ? m.e[j][i].im : m.e[i][j].im));
        }
}
template <typename T, int LAYOUT>
__device__ __forceinline__ Su3<T> load_mat(const T *__restrict__ f, size_t plane0, size_t Vh, size_t i)
{
    Su3<T> m;
    const L2Pol pol = {0, 0};
#pragma unroll
    for (int k = 0; k < 9; ++k) m.e[k / 3][k % 3] = ld_cx<T, LAYOUT, 0, 0>(f, plane0 + k, Vh, i, pol);
    return m;
}
template <typename T, int LAYOUT>
__device__ __forceinline__ void store_mat(T *__restrict__ f, size_t plane0, size_t Vh, size_t i, const Su3<T> &m)
{
    const L2Pol pol = {0, 0};
#pragma unroll
    for (int k = 0; k < 9; ++k) st_cx<T, LAYOUT, 0>(f, plane0 + k, Vh, i, m.e[k / 3][k % 3], pol);
}
// the staple field is written once and not read again by this library: streaming stores keep the link
// neighbourhood in L2 (ncu on variant 1: 855 MB written to DRAM against 604 MB of output)
template <typename T, int LAYOUT>
__device__ __forceinline__ void store_mat_stream(T *__restrict__ f, size_t plane0, size_t Vh, size_t i, const Su3<T> &m)
{
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const Cx<T> z = m.e[k / 3][k % 3];
        if (LAYOUT == 0) {
            typedef typename Vec2<T>::type V2;
            V2 v; v.x = z.re; v.y = z.im;
            __stcs(reinterpret_cast<V2 *>(f) + (plane0 + k) * Vh + i, v);
        } else {
            __stcs(f + (2 * (plane0 + k)) * Vh + i, z.re);
            __stcs(f + (2 * (plane0 + k) + 1) * Vh + i, z.im);
        }
    }
}

__device__ __forceinline__ Site4 decode_site(const Geom &g, int i, int parity)
{
    uint32_t t = fd_div((uint32_t)i, g.dNh0);
    const int hx0 = i - (int)t * g.Nh0;
    uint32_t t2 = fd_div(t, g.dN1);
    Site4 x;
    x.x1 = (int)t - (int)t2 * g.N1;
    x.x3 = (int)fd_div(t2, g.dN2);
    x.x2 = (int)t2 - x.x3 * g.N2;
    x.x0 = 2 * hx0 + ((x.x1 + x.x2 + x.x3 + parity) & 1);
    return x;
}

// Storage of the 48 intermediate fields (24 per parity).  TF_TILED 1: [field][tile of 128 sites][k = 0..8][site in tile] --
// the nine entries of a matrix of one tile are contiguous (18 KB in fp64), so that a CTA's accesses to one matrix fall
// into one DRAM page region and the entry offsets are compile-time constants; 0: nine planes of Vh sites per field,
// like the links.
#ifndef PRODUCE_MINB
#define PRODUCE_MINB 4      // (128,4): 128 registers, no spills; 2.568 -> 2.539 ns/site at 32^4 fp64 against (128,3)
#endif
#ifndef TF_TILED
#define TF_TILED 1
#endif
__host__ __device__ __forceinline__ size_t tf_sites(size_t Vh) { return TF_TILED ? (Vh + 127) / 128 * 128 : Vh; }
template <typename T, int LAYOUT>
__device__ __forceinline__ Su3<T> load_tmat(const T *__restrict__ f, size_t plane0, size_t Vh, size_t i)
{
    if (!TF_TILED) return load_mat<T, LAYOUT>(f, plane0, Vh, i);
    typedef typename Vec2<T>::type V2;
    const size_t base = ((plane0 / 9) * (tf_sites(Vh) / 128) + (i >> 7)) * (9 * 128) + (i & 127);    // in complex numbers
    Su3<T> m;
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        if (LAYOUT == 0) {
            const V2 v = __ldg(reinterpret_cast<const V2 *>(f) + base + k * 128);
            m.e[k / 3][k % 3] = cx<T>(v.x, v.y);
        } else {
            const T *p = f + 2 * (base - (i & 127)) + (2 * k) * 128 + (i & 127);
            m.e[k / 3][k % 3] = cx<T>(__ldg(p), __ldg(p + 128));
        }
    }
    return m;
}
template <typename T, int LAYOUT>
__device__ __forceinline__ void store_tmat(T *__restrict__ f, size_t plane0, size_t Vh, size_t i, const Su3<T> &m)
{
    if (!TF_TILED) { store_mat<T, LAYOUT>(f, plane0, Vh, i, m); return; }
    typedef typename Vec2<T>::type V2;
    const size_t base = ((plane0 / 9) * (tf_sites(Vh) / 128) + (i >> 7)) * (9 * 128) + (i & 127);
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const Cx<T> z = m.e[k / 3][k % 3];
        if (LAYOUT == 0) {
            V2 v; v.x = z.re; v.y = z.im;
            reinterpret_cast<V2 *>(f)[base + k * 128] = v;
        } else {
            T *p = f + 2 * (base - (i & 127)) + (2 * k) * 128 + (i & 127);
            p[0] = z.re; p[128] = z.im;
        }
    }
}

// Pass 1.  CTA = 128 consecutive sites of one parity; blockIdx.x = (tile * 2 + parity) * 12 + ordered pair, so
// that the 24 CTAs that read the links of one tile run together.
template <typename T, int LAYOUT, int RECON12>
__global__ void __launch_bounds__(128, PRODUCE_MINB) staples_produce_kernel(const Geom g, T *__restrict__ tf, const T *__restrict__ links)
{
    pdl_wait();
    pdl_trigger();
    const int bid = blockIdx.x;
    const int q = bid % 12, parity = (bid / 12) & 1, tile = bid / 24;
    const int i = tile * blockDim.x + threadIdx.x;
    if (i >= g.Vh) return;
    const int m = q / 3, n = (q % 3) + ((q % 3) >= m ? 1 : 0);
    const Site4 x = decode_site(g, i, parity);
    const size_t Vh = (size_t)g.Vh, Ls = (size_t)g.Ls;
    const size_t im = (size_t)(i + idxh_disp(g, x, m, 1)), in = (size_t)(i + idxh_disp(g, x, n, 1));
    const L2Pol pol = {0, 0};
    Su3<T> Q;
    {
        const Su3<T> a = load_link<T, LAYOUT, RECON12, 0, 0>(links, parity, m, Ls, (size_t)i, pol);
        const Su3<T> d = load_link<T, LAYOUT, RECON12, 0, 0>(links, parity ^ 1, n, Ls, im, pol);
        Q = mul_op<T, 0, 0>(a, d);                                      // U_m(y) U_n(y+m)
    }
    {
        const Su3<T> b = load_link<T, LAYOUT, RECON12, 0, 0>(links, parity, n, Ls, (size_t)i, pol);
        store_tmat<T, LAYOUT>(tf, tfield_plane(parity ^ 1, pair_idx(m, n), 1), Vh, in, mul_op<T, 1, 0>(Q, b));   // Tl_mn(y+n)
    }
    {
        const Su3<T> c = load_link<T, LAYOUT, RECON12, 0, 0>(links, parity ^ 1, m, Ls, in, pol);
        store_tmat<T, LAYOUT>(tf, tfield_plane(parity, pair_idx(n, m), 0), Vh, (size_t)i, mul_op<T, 0, 1>(c, Q)); // Tu_nm(y)
    }
}

// Pass 2.  One thread per link (x, mu); CTA order as in the one-pass kernels (staple_cta).
template <typename T, int LAYOUT, int RECON12, int MINB>
__global__ void __launch_bounds__(128, MINB) staples_final_kernel(const Geom g, T *__restrict__ staples, const T *__restrict__ links,
                                                             const T *__restrict__ tf, const T c0, const T c1, const StapleSwizzle sw)
{
    pdl_wait();
    pdl_trigger();
    int tile, mu, parity;
    staple_cta(sw, tile, mu, parity);
    const int i = tile * blockDim.x + threadIdx.x;
    if (i >= g.Vh) return;
    const Site4 x = decode_site(g, i, parity);
    const size_t Vh = (size_t)g.Vh, Ls = (size_t)g.Ls;
    const L2Pol pol = {0, 0};
    const int po = parity ^ 1;
    const size_t i_m = (size_t)(i + idxh_disp(g, x, mu, 1));           // x + mu
    Su3<T> S;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) S.e[a][b] = cx<T>((T)0, (T)0);
#pragma unroll 1
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        const int dn_p = idxh_disp(g, x, nu, 1), dn_m = idxh_disp(g, x, nu, -1);
        const size_t i_n = (size_t)(i + dn_p), i_l = (size_t)(i + dn_m);                       // x + nu, x - nu
        const size_t i_ml = (size_t)((int)i_m + dn_m);                                           // x + mu - nu
        const int qmn = pair_idx(mu, nu), qnm = pair_idx(nu, mu);
        // (prefetching the next nu's stored staples / links into L2 from here was tried: 2.63 -> 2.68 / 2.83 ns/site at 32^4
        // fp64 -- the kernel is not waiting for DRAM alone; profiles/sweep_r2.md section 3)
        // c0 Tu_munu(x) = c0 (A B) C and c0 Tl_munu(x) = c0 (A' B') C' are folded into the (A B) products, so the
        // link's own two staple fields are not loaded: 6 matrix loads and 5 products per half.
        {   // above the link
            const Su3<T> Ub = load_link<T, LAYOUT, RECON12, 0, 0>(links, po, mu, Ls, i_n, pol);           // U_mu(x+nu)
            const Su3<T> A = load_link<T, LAYOUT, RECON12, 0, 0>(links, po, nu, Ls, i_m, pol);            // U_nu(x+mu)
            Su3<T> W;
            {
                const Su3<T> T1 = load_tmat<T, LAYOUT>(tf, tfield_plane(po, qnm, 0), Vh, i_m);             // Tu_numu(x+mu)
                W = mul_op<T, 1, 1>(T1, Ub);                                                                // T1^+ B
            }
            {
                const Su3<T> T2 = load_tmat<T, LAYOUT>(tf, tfield_plane(po, qmn, 0), Vh, i_n);             // Tu_munu(x+nu)
                acc_op<T, 0>(W, (T)1, mul_op<T, 0, 0>(A, T2));
            }
            const Su3<T> AB = mul_op<T, 0, 1>(A, Ub);
            const Su3<T> Uc = load_link<T, LAYOUT, RECON12, 0, 0>(links, parity, nu, Ls, (size_t)i, pol); // U_nu(x)
            {
                Su3<T> X = load_tmat<T, LAYOUT>(tf, tfield_plane(parity, qnm, 1), Vh, (size_t)i);          // Tl_numu(x)
                scale_acc_op<T, 1>(X, c1, c0, Uc);                                                          // c1 T3 + c0 C
                acc_op<T, 0>(S, (T)1, mul_op<T, 0, 0>(AB, X));
            }
            acc_op<T, 0>(S, c1, mul_op<T, 0, 1>(W, Uc));
        }
        {   // below the link
            const Su3<T> Ub = load_link<T, LAYOUT, RECON12, 0, 0>(links, po, mu, Ls, i_l, pol);           // U_mu(x-nu)
            const Su3<T> Ua = load_link<T, LAYOUT, RECON12, 0, 0>(links, parity, nu, Ls, i_ml, pol);      // U_nu(x+mu-nu)
            Su3<T> W;
            {
                const Su3<T> T1 = load_tmat<T, LAYOUT>(tf, tfield_plane(parity, qnm, 0), Vh, i_ml);        // Tu_numu(x+mu-nu)
                W = mul_op<T, 0, 1>(T1, Ub);
            }
            {
                const Su3<T> T2 = load_tmat<T, LAYOUT>(tf, tfield_plane(po, qmn, 1), Vh, i_l);             // Tl_munu(x-nu)
                acc_op<T, 0>(W, (T)1, mul_op<T, 1, 0>(Ua, T2));
            }
            const Su3<T> AB = mul_op<T, 1, 1>(Ua, Ub);
            const Su3<T> Uc = load_link<T, LAYOUT, RECON12, 0, 0>(links, po, nu, Ls, i_l, pol);           // U_nu(x-nu)
            {
                const Su3<T> T3 = load_tmat<T, LAYOUT>(tf, tfield_plane(po, qnm, 1), Vh, i_l);             // Tl_numu(x-nu)
                Su3<T> X;                                                                                   // c1 T3^+ + c0 C'
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b)
                        X.e[a][b] = cx<T>(fma(c1, T3.e[b][a].re, c0 * Uc.e[a][b].re), fma(-c1, T3.e[b][a].im, c0 * Uc.e[a][b].im));
                acc_op<T, 0>(S, (T)1, mul_op<T, 0, 0>(AB, X));
            }
            acc_op<T, 0>(S, c1, mul_op<T, 0, 0>(W, Uc));
        }
    }
    store_mat_stream<T, LAYOUT>(staples, (size_t)((parity * 4 + mu) * 9), Vh, (size_t)i, S);
}

extern "C" size_t lqcd_staples_workspace_bytes(const lqcd_ctx *ctx)
{
    return ctx ? tf_sites((size_t)ctx->g.Vh) * 2 * 24 * 9 * 2 * elem_size(ctx) : 0;
}

extern "C" int lqcd_gauge_staples(lqcd_ctx *ctx, const void *links, void *staples, double c0, double c1)
{
    if (!ctx) return LQCD_ERR_ARG;
    int rc = lqcd_check_cuda(ctx, cudaSetDevice(ctx->device), "cudaSetDevice");
    if (rc) return rc;
    if (!links || !staples) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_gauge_staples: null pointer");
    if (links == staples) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_gauge_staples: staples alias links");
    if (c0 != c0 || c1 != c1) return lqcd_fail(ctx, LQCD_ERR_ARG, "lqcd_gauge_staples: NaN coefficient");
    if (ctx->halo_fn || ctx->x3_lo != 0 || ctx->x3_hi != ctx->g.N3)
        return lqcd_fail(ctx, LQCD_ERR_UNSUPPORTED, "lqcd_gauge_staples: not available in slab mode (second-neighbour halo)");
    dim3 grid(((ctx->g.Vh + 127) / 128) * 8), block(128);
    StapleSwizzle sw = {0, 0, ctx->g.N2, ctx->g.N3};
    const int row = ctx->g.Nh0 * ctx->g.N1;          // half-sites per (x2, x3) row
    if (ctx->staples_x2block > 0 && row % 128 == 0 && ctx->g.N2 % ctx->staples_x2block == 0) {
        sw.x2b = ctx->staples_x2block;
        sw.tiles_row = row / 128;
    }
    // variant 2 needs the intermediate fields in the context's workspace; without one that is large enough the
    // one-pass kernel with shared sub-products runs instead (same result to rounding)
    const bool two_pass = ctx->staples_variant == 2 && ctx->ws && ctx->ws_bytes >= lqcd_staples_workspace_bytes(ctx);
    ctx->staples_ran = two_pass ? 2 : (ctx->staples_variant == 0 ? 0 : 1);
    if (two_pass) {
        dim3 gridp(((ctx->g.Vh + 127) / 128) * 24);
        int minb = ctx->staples_minblocks;           // launch-bounds variant of pass 2 (0: default per precision)
        if (minb == 0) minb = ctx->prec == LQCD_F64 ? 2 : 4;      // measured best: profiles/sweep_r2.md section 3
#define GO2(T, L, R) do { \
        launch_k(ctx, staples_produce_kernel<T, L, R>, gridp, block, ctx->g, (T *)ctx->ws, (const T *)links); \
        if (minb == 2) launch_k(ctx, staples_final_kernel<T, L, R, 2>, grid, block, ctx->g, (T *)staples, (const T *)links, (const T *)ctx->ws, (T)c0, (T)c1, sw); \
        else if (minb == 3) launch_k(ctx, staples_final_kernel<T, L, R, 3>, grid, block, ctx->g, (T *)staples, (const T *)links, (const T *)ctx->ws, (T)c0, (T)c1, sw); \
        else launch_k(ctx, staples_final_kernel<T, L, R, 4>, grid, block, ctx->g, (T *)staples, (const T *)links, (const T *)ctx->ws, (T)c0, (T)c1, sw); } while (0)
#define GO2R(T, L) do { if (ctx->recon == LQCD_RECON_12) GO2(T, L, 1); else GO2(T, L, 0); } while (0)
        if (ctx->prec == LQCD_F64) { if (ctx->layout == 0) GO2R(double, 0); else GO2R(double, 1); }
        else { if (ctx->layout == 0) GO2R(float, 0); else GO2R(float, 1); }
#undef GO2R
#undef GO2
        return lqcd_check_cuda(ctx, cudaGetLastError(), "gauge staples (two passes)");
    }
#define GO(T, L) do { \
        if (ctx->staples_variant >= 1) { \
            if (ctx->recon == LQCD_RECON_12) launch_k(ctx, staples_kernel_shared<T, L, 1>, grid, block, ctx->g, (T *)staples, (const T *)links, (T)c0, (T)c1, sw); \
            else launch_k(ctx, staples_kernel_shared<T, L, 0>, grid, block, ctx->g, (T *)staples, (const T *)links, (T)c0, (T)c1, sw); \
        } else if (ctx->recon == LQCD_RECON_12) launch_k(ctx, staples_kernel<T, L, 1>, grid, block, ctx->g, (T *)staples, (const T *)links, (T)c0, (T)c1, sw); \
        else launch_k(ctx, staples_kernel<T, L, 0>, grid, block, ctx->g, (T *)staples, (const T *)links, (T)c0, (T)c1, sw); } while (0)
    if (ctx->prec == LQCD_F64) { if (ctx->layout == 0) GO(double, 0); else GO(double, 1); }
    else { if (ctx->layout == 0) GO(float, 0); else GO(float, 1); }
#undef GO
    return lqcd_check_cuda(ctx, cudaGetLastError(), "gauge staples");
}
