// su3.cuh -- link and colour-vector loads shared by the stencil kernels (dslash.cu, force.cu):
// step a3 of SURVEY.md section 8(a) (link fetch with streaming loads, optional third-row rebuild
// r2 = (r0 ^ r1)^*, reading R8).
#pragma once
#include "common.cuh"

template <typename T> struct Su3 { Cx<T> e[3][3]; };

// STREAM = 1: evict-first loads (each link read once: Dslash, force); 0: cached loads (staples re-read
// every link ~100 times from L1/L2).
template <typename T, int LAYOUT, int RECON12, int POLICY, int STREAM = 1>
__device__ __forceinline__ Su3<T> load_link(const T *__restrict__ links, int par, int mu, size_t Vh, size_t i, const L2Pol &pol)
{
    constexpr int R = RECON12 ? 2 : 3;
    Su3<T> u;
    size_t plane0 = (size_t)(par * 4 + mu) * (R * 3);
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) u.e[r][c] = ld_cx<T, LAYOUT, STREAM, POLICY>(links, plane0 + r * 3 + c, Vh, i, pol);
    if (RECON12) {
        // r2[k] = conj( eps_kij r0[i] r1[j] )   (reading R8)
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int a = (k + 1) % 3, b = (k + 2) % 3;
            Cx<T> x = u.e[0][a], y = u.e[1][b], z = u.e[0][b], w = u.e[1][a];
            T re = x.re * y.re - x.im * y.im - (z.re * w.re - z.im * w.im);
            T im = x.re * y.im + x.im * y.re - (z.re * w.im + z.im * w.re);
            u.e[2][k] = cx<T>(re, -im);
        }
    }
    return u;
}

// acc += U p
template <typename T> __device__ __forceinline__ void mv_acc(Cx<T> acc[3], const Su3<T> &u, const Cx<T> p[3])
{
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            acc[a].re = fma(u.e[a][b].re, p[b].re, acc[a].re);
            acc[a].re = fma(-u.e[a][b].im, p[b].im, acc[a].re);
            acc[a].im = fma(u.e[a][b].re, p[b].im, acc[a].im);
            acc[a].im = fma(u.e[a][b].im, p[b].re, acc[a].im);
        }
}
// acc += U^dagger p,  (U^dagger)_{ab} = conj(U_{ba})
template <typename T> __device__ __forceinline__ void mvdag_acc(Cx<T> acc[3], const Su3<T> &u, const Cx<T> p[3])
{
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            acc[a].re = fma(u.e[b][a].re, p[b].re, acc[a].re);
            acc[a].re = fma(u.e[b][a].im, p[b].im, acc[a].re);
            acc[a].im = fma(u.e[b][a].re, p[b].im, acc[a].im);
            acc[a].im = fma(-u.e[b][a].im, p[b].re, acc[a].im);
        }
}

template <typename T, int LAYOUT, int POLICY>
__device__ __forceinline__ void load_vec(const T *__restrict__ v, size_t Vh, size_t i, T coef, Cx<T> p[3], const L2Pol &pol)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        Cx<T> z = ld_cx<T, LAYOUT, 0, POLICY>(v, (size_t)c, Vh, i, pol);
        p[c] = cx<T>(coef * z.re, coef * z.im);
    }
}

// p = coef * e^{i theta} * v(i): the backfield phase of a hop (reading R6) folded into the
// neighbour vector together with eta / the boundary sign.
__device__ __forceinline__ void sincos_t(double x, double *s, double *c) { sincos(x, s, c); }
__device__ __forceinline__ void sincos_t(float x, float *s, float *c) { sincosf(x, s, c); }
template <typename T, int LAYOUT, int POLICY>
__device__ __forceinline__ void load_vec_phase(const T *__restrict__ v, size_t Vh, size_t i, T coef, T theta, Cx<T> p[3], const L2Pol &pol)
{
    T sn, cs;
    sincos_t(theta, &sn, &cs);
    const T cr = coef * cs, ci = coef * sn;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        Cx<T> z = ld_cx<T, LAYOUT, 0, POLICY>(v, (size_t)c, Vh, i, pol);
        p[c] = cx<T>(cr * z.re - ci * z.im, cr * z.im + ci * z.re);
    }
}
// as load_vec_phase with the unit complex number (cos theta, sin theta) stored: conj = -1 takes e^{-i theta}
template <typename T, int LAYOUT, int POLICY>
__device__ __forceinline__ void load_vec_unit(const T *__restrict__ v, size_t Vh, size_t i, T coef, T conj, const T *__restrict__ bf,
                                              size_t k, Cx<T> p[3], const L2Pol &pol)
{
    typedef typename Vec2<T>::type V2;
    const V2 e = __ldcs(reinterpret_cast<const V2 *>(bf) + k);
    const T cr = coef * e.x, ci = coef * conj * e.y;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        Cx<T> z = ld_cx<T, LAYOUT, 0, POLICY>(v, (size_t)c, Vh, i, pol);
        p[c] = cx<T>(cr * z.re - ci * z.im, cr * z.im + ci * z.re);
    }
}
// a face vector from a landing buffer of the peer transport (peer.cuh): written by another GPU during this kernel's
// lifetime (before its flag), so it is read through L2 (ld.global.cg), never through the non-coherent path
// (cr, ci): the hop's coefficient times the backfield phase (ci = 0 without a backfield)
template <typename T, int LAYOUT>
__device__ __forceinline__ void load_vec_cg(const T *__restrict__ buf, size_t stride, size_t f, T cr, T ci, Cx<T> p[3])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        T re, im;
        if (LAYOUT == 0) {
            typedef typename Vec2<T>::type V2;
            const V2 v = __ldcg(reinterpret_cast<const V2 *>(buf) + (size_t)c * stride + f);
            re = v.x; im = v.y;
        } else {
            re = __ldcg(buf + (size_t)(2 * c) * stride + f); im = __ldcg(buf + (size_t)(2 * c + 1) * stride + f);
        }
        p[c] = cx<T>(cr * re - ci * im, cr * im + ci * re);
    }
}
// coef * e^{+-i theta} of link k of the native backfield (BF 1: theta stored, BF 2: (cos, sin) stored; conj = -1: e^{-i theta})
template <typename T, int BF>
__device__ __forceinline__ void phase_coef(const T *__restrict__ bf, size_t k, T coef, T conj, T *cr, T *ci)
{
    if (BF == 0) { *cr = coef; *ci = (T)0; return; }
    T sn, cs;
    if (BF == 1) sincos_t(__ldcs(bf + k), &sn, &cs);
    else { cs = __ldcs(bf + 2 * k); sn = __ldcs(bf + 2 * k + 1); }
    *cr = coef * cs; *ci = coef * conj * sn;
}
