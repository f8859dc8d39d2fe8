// dwf_aux.cuh -- everything on the path that is not the stencil: layout reorder (a1), the closed-form
// M_oo^{-1} (a5), BLAS-1 with fp64 reductions (a7) and the fused CG vector updates (a9).
#pragma once
#include "dwf_vec.cuh"

namespace dwf {

// ------------------------------------------------------------------------------------------------
// a1. canonical <-> native reorder.  canonical spinor: complex<R> [nrhs][Ls][V4 lex][12];
// native: group index ((blk_index(site, r)*12 + c)*K + k), K = Ls/VL, group k holds lanes s = k*VL .. k*VL+VL-1.
// ------------------------------------------------------------------------------------------------
// One warp per (site, rhs) block, staged through shared memory: the canonical side moves in 96R-byte runs (the 12 complex
// components of one (s, site)), the native side in whole 16-byte groups of the contiguous block -- full sectors both ways.
// blockIdx.y = parity slot; dynamic shared memory = (warps per CTA) x 24 Ls reals.
template <typename R, bool IMPORT>
__global__ void __launch_bounds__(128)
reorder_spinor_kernel(const R* __restrict__ canon_in, R* __restrict__ canon_out,
                      typename Prec<R>::G* native0, typename Prec<R>::G* native1,
                      const int* __restrict__ lex0, const int* __restrict__ lex1,
                      long long V4h, long long V4, int Ls, int nrhs, int sg_shift, long long wid0, long long wid1) {
    using G = typename Prec<R>::G;
    constexpr int VL = Prec<R>::VL;
    extern __shared__ __align__(16) unsigned char smem_reorder[];
    const int K = Ls / VL, NG = 12 * K;                         // groups per block
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    R* buf = reinterpret_cast<R*>(smem_reorder) + (size_t)warp * 24 * Ls;
    const long long wid = wid0 + (long long)blockIdx.x * (blockDim.x >> 5) + warp;   // (site, rhs) pair of this parity, in [wid0, wid1)
    if (wid >= wid1) return;                                     // whole warps leave together
    const long long site = wid / nrhs;
    const int r = (int)(wid - site * nrhs);
    G* native = (blockIdx.y ? native1 : native0) + (size_t)blk_index(site, r, nrhs, sg_shift) * NG;
    const long long lx = (blockIdx.y ? lex1 : lex0)[site];
    // position of the real (s, c, reim) inside the native block, in reals
    auto npos = [&](int s, int c, int reim) -> int {
        if constexpr (VL == 2) return ((c * K + (s >> 1)) << 2) + (reim << 1) + (s & 1);
        else                   return ((c * K + s) << 1) + reim;
    };
    if constexpr (IMPORT) {
        for (int idx = lane; idx < Ls * 12; idx += 32) {         // idx = s*12 + c: one complex number per lane, 12 lanes per 96R-byte run
            const int s = idx / 12, c = idx - s * 12;
            const size_t ci = ((((size_t)r * Ls + s) * V4 + lx) * 12 + c) * 2;
            buf[npos(s, c, 0)] = canon_in[ci]; buf[npos(s, c, 1)] = canon_in[ci + 1];
        }
        __syncwarp();
        const G* bg = reinterpret_cast<const G*>(buf);
        for (int g = lane; g < NG; g += 32) native[g] = bg[g];
    } else {
        G* bg = reinterpret_cast<G*>(buf);
        for (int g = lane; g < NG; g += 32) bg[g] = native[g];
        __syncwarp();
        for (int idx = lane; idx < Ls * 12; idx += 32) {
            const int s = idx / 12, c = idx - s * 12;
            const size_t ci = ((((size_t)r * Ls + s) * V4 + lx) * 12 + c) * 2;
            canon_out[ci] = buf[npos(s, c, 0)]; canon_out[ci + 1] = buf[npos(s, c, 1)];
        }
    }
}

// canonical gauge complex<R> [mu][V4 lex][9] -> native [parity][V4h][mu][18]; U_t on the last time
// slice is stored with the antiperiodic sign (R3).
template <typename R>
__global__ void reorder_gauge_kernel(const R* __restrict__ canon, R* __restrict__ native,
                                     const int* __restrict__ lex /*[2][V4h]*/, long long V4h, long long V4,
                                     long long spatial /*Lx*Ly*Lz*/, int Lt) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= 2 * V4h * 4 * 9) return;
    const int k = (int)(gid % 9);
    const int mu = (int)((gid / 9) % 4);
    const long long ps = gid / 36;                          // p*V4h + site
    const long long lx = lex[ps];
    const R sign = (mu == 3 && lx / spatial == Lt - 1) ? R(-1) : R(1);
    const size_t ci = (((size_t)mu * V4 + lx) * 9 + k) * 2;
    native[gid * 2] = sign * canon[ci];
    native[gid * 2 + 1] = sign * canon[ci + 1];
}

// Precision conversion between the native layouts of two handles on the same lattice (mixed-precision solve).  The two
// handles may order their sites differently (tile shape depends on the precision): inv_src[lexicographic site] = index of
// that site in the source order of its parity, lex_dst[parity][site] = lexicographic site of the destination order.
__global__ void invert_lex_kernel(const int* __restrict__ lex /*[2][V4h]*/, int* __restrict__ inv /*[V4]*/, long long V4h) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= 2 * V4h) return;
    inv[lex[gid]] = (int)(gid % V4h);
}
// one thread per (destination block, component c, pair of s): handles s = 2j, 2j+1
template <typename RS, typename RD>
__global__ void convert_kernel(const typename Prec<RS>::G* __restrict__ src, typename Prec<RD>::G* __restrict__ dst,
                               const int* __restrict__ inv_src, const int* __restrict__ lex_dst, long long V4h,
                               int Ls, int nrhs, int sg_src, int sg_dst, int parities) {
    const int KP = Ls / 2;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = (long long)parities * V4h * nrhs * 12 * KP;
    if (gid >= total) return;
    const int j = (int)(gid % KP);
    const int c = (int)((gid / KP) % 12);
    const int r = (int)((gid / (12 * KP)) % nrhs);
    const long long ps = gid / ((long long)12 * KP * nrhs);           // p * V4h + destination site
    const long long p = ps / V4h, sd = ps - p * V4h;
    const long long ss = inv_src[lex_dst[ps]];
    const size_t half_s = (size_t)V4h * nrhs * 12 * (Ls / Prec<RS>::VL), half_d = (size_t)V4h * nrhs * 12 * (Ls / Prec<RD>::VL);
    const size_t bs = (size_t)blk_index(ss, r, nrhs, sg_src), bd = (size_t)blk_index(sd, r, nrhs, sg_dst);
    double re0, im0, re1, im1;
    if constexpr (Prec<RS>::VL == 2) {
        const float4 g = src[p * half_s + (bs * 12 + c) * KP + j];
        re0 = g.x; re1 = g.y; im0 = g.z; im1 = g.w;
    } else {
        const double2 g0 = src[p * half_s + (bs * 12 + c) * Ls + 2 * j], g1 = src[p * half_s + (bs * 12 + c) * Ls + 2 * j + 1];
        re0 = g0.x; im0 = g0.y; re1 = g1.x; im1 = g1.y;
    }
    if constexpr (Prec<RD>::VL == 2) {
        dst[p * half_d + (bd * 12 + c) * KP + j] = make_float4((float)re0, (float)re1, (float)im0, (float)im1);
    } else {
        dst[p * half_d + (bd * 12 + c) * Ls + 2 * j] = make_double2(re0, im0);
        dst[p * half_d + (bd * 12 + c) * Ls + 2 * j + 1] = make_double2(re1, im1);
    }
}

// Gathered links for the tiled stencil (dwf_tile.cuh): per site [mu][U_mu(x) 18 | U_mu(x-mu) 18] + padding,
// pre-scaled by -1/2 (exact), so that a tile's links are one contiguous run and need no index lookup.
template <typename R>
__global__ void gather_links_kernel(const R* __restrict__ gauge /*[2][V4h][4][18]*/, R* __restrict__ glinks /*[2][V4h][site_reals]*/,
                                    const int* __restrict__ nbr /*[2][V4h][8]*/, long long V4h, int site_reals) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= 2 * V4h * 4 * 36) return;
    const int j = (int)(gid % 36);
    const int mu = (int)((gid / 36) % 4);
    const long long ps = gid / 144;                         // p*V4h + site
    R v;
    if (j < 18) v = gauge[(ps * 4 + mu) * 18 + j];
    else {
        const long long p = ps / V4h;
        const long long q = (1 - p) * V4h + nbr[ps * 8 + 2 * mu + 1];
        v = gauge[(q * 4 + mu) * 18 + (j - 18)];
    }
    glinks[ps * site_reals + mu * 36 + j] = R(-0.5) * v;
}

// ------------------------------------------------------------------------------------------------
// a5. Exact inverse of the 4D-site-diagonal block M_oo = M_ee.  Per site, per
// complex component, per rhs the Ls x Ls system is cyclic bidiagonal:
//    d v_j - v_{j-1} = b_j (j >= 1),   d v_0 + m v_{Ls-1} = b_0      (j = s for the P_+ half,
//                                                                     j = Ls-1-s for the P_- half;
//                                                                     adjoint: halves swapped)
// solved exactly by   w_0 = 0, w_j = k (b_j + w_{j-1});  v_0 = k (b_0 - m w_{Ls-1}) / (1 + m k^Ls);
//                     v_j = w_j + k^j v_0,               k = 1/d = 1/(5 - M5).
// One thread per (site, component, rhs) walks s in registers.  In place is allowed.
// ------------------------------------------------------------------------------------------------
template <typename R, int LS, bool DAG>
__global__ void __launch_bounds__(128)
mooinv_kernel(const typename Prec<R>::G* in, typename Prec<R>::G* out, long long V4h, int nrhs, int sg_shift,
              R kappa, R mass, R v0scale /* kappa / (1 + m kappa^Ls) */) {
    using G = typename Prec<R>::G;
    constexpr int VL = Prec<R>::VL;
    constexpr int NG = LS / VL;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= V4h * 12 * nrhs) return;
    const int r = (int)(gid % nrhs);
    const int c = (int)((gid / nrhs) % 12);
    const long long site = gid / (12 * nrhs);
    const size_t base = ((size_t)blk_index(site, r, nrhs, sg_shift) * 12 + c) * NG;
    const bool down = DAG ? (c >= 6) : (c < 6);
    R bre[LS], bim[LS];
#pragma unroll
    for (int k = 0; k < NG; k++) {
        const G g = in[base + (down ? k : NG - 1 - k)];
        if constexpr (VL == 2) {
            bre[2 * k] = down ? g.x : g.y; bre[2 * k + 1] = down ? g.y : g.x;
            bim[2 * k] = down ? g.z : g.w; bim[2 * k + 1] = down ? g.w : g.z;
        } else { bre[k] = g.x; bim[k] = g.y; }
    }
    const R b0re = bre[0], b0im = bim[0];
    bre[0] = R(0); bim[0] = R(0);
#pragma unroll
    for (int j = 1; j < LS; j++) { bre[j] = kappa * (bre[j] + bre[j - 1]); bim[j] = kappa * (bim[j] + bim[j - 1]); }
    const R v0re = v0scale * (b0re - mass * bre[LS - 1]);
    const R v0im = v0scale * (b0im - mass * bim[LS - 1]);
    R pw = R(1);
#pragma unroll
    for (int j = 0; j < LS; j++) { bre[j] = fma(pw, v0re, bre[j]); bim[j] = fma(pw, v0im, bim[j]); pw *= kappa; }
#pragma unroll
    for (int k = 0; k < NG; k++) {
        G g;
        if constexpr (VL == 2) {
            g.x = down ? bre[2 * k] : bre[2 * k + 1]; g.y = down ? bre[2 * k + 1] : bre[2 * k];
            g.z = down ? bim[2 * k] : bim[2 * k + 1]; g.w = down ? bim[2 * k + 1] : bim[2 * k];
        } else { g.x = bre[k]; g.y = bim[k]; }
        out[base + (down ? k : NG - 1 - k)] = g;
    }
}

// ------------------------------------------------------------------------------------------------
// a7. BLAS-1.  Fields are flat arrays of groups; group e belongs to rhs (e / BS) % nrhs, BS = groups per
// run of one rhs (12*Ls/VL groups per (site, rhs) block x sites per site group).  Launch geometry guarantees (gridDim.x * blockDim.x) % (BS*nrhs) == 0,
// so a thread keeps one rhs for its whole grid-stride loop.  Reductions: fp64 per-thread accumulation, fixed-
// order in-block combine per rhs, per-block partials, fixed-order final pass => deterministic.
// ------------------------------------------------------------------------------------------------
struct RhsCoef { double re[64]; double im[64]; };

template <typename R>
__global__ void axpy_kernel(const typename Prec<R>::G* __restrict__ x, typename Prec<R>::G* y,
                            long long ngroups, int BS, int nrhs, RhsCoef a) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int r = (int)((e / BS) % nrhs);
    const R are = (R)a.re[r], aim = (R)a.im[r];
    for (; e < ngroups; e += stride) {
        const CV<V> xx = unpack(ldg_nc(x + e));
        CV<V> yy = unpack(y[e]);
        yy.re = vfnma(aim, xx.im, vfma(are, xx.re, yy.re));
        yy.im = vfma(aim, xx.re, vfma(are, xx.im, yy.im));
        y[e] = pack(yy);
    }
}

__device__ __forceinline__ void acc_inner(double& sre, double& sim, CV<float2> x, CV<float2> y) {
    sre += (double)x.re.x * y.re.x + (double)x.im.x * y.im.x + (double)x.re.y * y.re.y + (double)x.im.y * y.im.y;
    sim += (double)x.re.x * y.im.x - (double)x.im.x * y.re.x + (double)x.re.y * y.im.y - (double)x.im.y * y.re.y;
}
__device__ __forceinline__ void acc_inner(double& sre, double& sim, CV<double> x, CV<double> y) {
    sre += x.re * y.re + x.im * y.im;
    sim += x.re * y.im - x.im * y.re;
}

// Fixed-order combine of the 256 per-thread sums of a block into per-rhs block partials
// partial[(blockIdx.x * nrhs + r) * 2 + {0,1}]  (north_star item (4): warp shuffle + block reduction).
// When the groups of one rhs come in runs that are a multiple of 32 (BS % 32 == 0: every production layout) all lanes of a warp
// hold the same rhs: a butterfly of shuffles reduces the warp, and thread r adds the (at most 8) warp sums of its rhs in warp
// order.  Otherwise (narrow blocks of the generic layout) thread r walks the 256 entries of its rhs in thread order.
__device__ __forceinline__ void block_combine(double sre, double sim, int r, int nrhs, int BS, double* partial) {
    __shared__ double s_re[256], s_im[256];
    __shared__ int s_r[256];
    const int t = threadIdx.x;
    if ((BS & 31) == 0) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            sre += __shfl_xor_sync(0xffffffffu, sre, off);
            sim += __shfl_xor_sync(0xffffffffu, sim, off);
        }
        if ((t & 31) == 0) { s_re[t >> 5] = sre; s_im[t >> 5] = sim; s_r[t >> 5] = r; }
        __syncthreads();
        if (t < nrhs) {
            double a = 0, b = 0;
            const int nw = (int)blockDim.x >> 5;
            for (int w = 0; w < nw; w++) if (s_r[w] == t) { a += s_re[w]; b += s_im[w]; }
            partial[((size_t)blockIdx.x * nrhs + t) * 2] = a;
            partial[((size_t)blockIdx.x * nrhs + t) * 2 + 1] = b;
        }
        return;
    }
    s_re[t] = sre; s_im[t] = sim; s_r[t] = r;
    __syncthreads();
    if (t < nrhs) {
        double a = 0, b = 0;
        for (int q = 0; q < (int)blockDim.x; q++) if (s_r[q] == t) { a += s_re[q]; b += s_im[q]; }
        partial[((size_t)blockIdx.x * nrhs + t) * 2] = a;
        partial[((size_t)blockIdx.x * nrhs + t) * 2 + 1] = b;
    }
}

template <typename R, bool NORM>
__global__ void __launch_bounds__(256)
inner_kernel(const typename Prec<R>::G* __restrict__ x, const typename Prec<R>::G* __restrict__ y,
             long long ngroups, int BS, int nrhs, double* partial) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int r = (int)((e / BS) % nrhs);
    double sre = 0, sim = 0;
    for (; e < ngroups; e += stride) {
        const CV<V> xx = unpack(ldg_nc(x + e));
        if constexpr (NORM) acc_inner(sre, sim, xx, xx);
        else                acc_inner(sre, sim, xx, unpack(ldg_nc(y + e)));
    }
    block_combine(sre, sim, r, nrhs, BS, partial);
}

// out[r*ostride + {0,1}] = sum over blocks of partial.  One block of 256 threads per rhs: thread t adds the partials
// t, t+256, ... in that order, then a fixed binary tree combines the 256 sums: deterministic, and ~100x faster than
// one thread walking all the partials.
__global__ void __launch_bounds__(256)
reduce_final_kernel(const double* __restrict__ partial, int nblocks, int nrhs, double* out, int ostride, int ncomp) {
    __shared__ double s_a[256], s_b[256];
    const int r = blockIdx.x, t = threadIdx.x;
    double a = 0, b = 0;
    for (int k = t; k < nblocks; k += 256) { a += partial[((size_t)k * nrhs + r) * 2]; b += partial[((size_t)k * nrhs + r) * 2 + 1]; }
    s_a[t] = a; s_b[t] = b;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (t < w) { s_a[t] += s_a[t + w]; s_b[t] += s_b[t + w]; }
        __syncthreads();
    }
    if (t == 0) { out[r * ostride] = s_a[0]; if (ncomp > 1) out[r * ostride + 1] = s_b[0]; }
}

// ------------------------------------------------------------------------------------------------
// a9. CG vector updates (half fields, nrhs right-hand sides: one CG per rhs in lock step), scalars read from device
// memory, one per rhs; launch geometry as for BLAS-1 (a thread keeps one rhs):
//   init  : r = b - q ; p = r ;                              partial |r|^2
//   xr    : alpha = rr[r] / pAp[r] ; x += alpha p ; r -= alpha q ; partial |r|^2
//   p     : beta  = rr_new[r] / rr_old[r] ; p = r + beta p
// ------------------------------------------------------------------------------------------------
template <typename R>
__global__ void __launch_bounds__(256)
cg_init_kernel(const typename Prec<R>::G* __restrict__ b, const typename Prec<R>::G* __restrict__ q,
               typename Prec<R>::G* r, typename Prec<R>::G* p, long long ngroups, int BS, int nrhs, double* partial) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int rhs = (int)((e / BS) % nrhs);
    double sre = 0, sim = 0;
    for (; e < ngroups; e += stride) {
        const CV<V> rr = csub(unpack(ldg_nc(b + e)), unpack(ldg_nc(q + e)));
        r[e] = pack(rr); p[e] = pack(rr);
        acc_inner(sre, sim, rr, rr);
    }
    block_combine(sre, sim, rhs, nrhs, BS, partial);
}

template <typename R>
__global__ void __launch_bounds__(256)
cg_update_xr_kernel(typename Prec<R>::G* x, typename Prec<R>::G* r, const typename Prec<R>::G* __restrict__ p,
                    const typename Prec<R>::G* __restrict__ q, long long ngroups, int BS, int nrhs,
                    const double* __restrict__ rr, const double* __restrict__ pAp, double* partial) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int rhs = (int)((e / BS) % nrhs);
    const R alpha = pAp[rhs] != 0.0 ? (R)(rr[rhs] / pAp[rhs]) : R(0);       // zero or converged right-hand side: frozen
    double sre = 0, sim = 0;
    for (; e < ngroups; e += stride) {
        const CV<V> pp = unpack(ldg_nc(p + e)), qq = unpack(ldg_nc(q + e));
        CV<V> xx = unpack(x[e]), rv = unpack(r[e]);
        xx.re = vfma(alpha, pp.re, xx.re); xx.im = vfma(alpha, pp.im, xx.im);
        rv.re = vfnma(alpha, qq.re, rv.re); rv.im = vfnma(alpha, qq.im, rv.im);
        x[e] = pack(xx); r[e] = pack(rv);
        acc_inner(sre, sim, rv, rv);
    }
    block_combine(sre, sim, rhs, nrhs, BS, partial);
}

// fused iteration (dwf_api.cu cg_t): x += alpha p ; p = r + beta p   (r already updated by the adjoint Schur launch)
template <typename R>
__global__ void __launch_bounds__(256)
cg_update_xp_kernel(typename Prec<R>::G* x, typename Prec<R>::G* p, const typename Prec<R>::G* __restrict__ r,
                    long long ngroups, int BS, int nrhs, const double* __restrict__ rr_old, const double* __restrict__ pAp,
                    const double* __restrict__ rr_new) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int rhs = (int)((e / BS) % nrhs);
    const R alpha = pAp[rhs] != 0.0 ? (R)(rr_old[rhs] / pAp[rhs]) : R(0);
    const R beta = rr_old[rhs] != 0.0 ? (R)(rr_new[rhs] / rr_old[rhs]) : R(0);
    for (; e < ngroups; e += stride) {
        const CV<V> rv = unpack(ldg_nc(r + e));
        CV<V> pp = unpack(p[e]), xx = unpack(x[e]);
        xx.re = vfma(alpha, pp.re, xx.re); xx.im = vfma(alpha, pp.im, xx.im);
        pp.re = vfma(beta, pp.re, rv.re); pp.im = vfma(beta, pp.im, rv.im);
        x[e] = pack(xx); p[e] = pack(pp);
    }
}

template <typename R>
__global__ void __launch_bounds__(256)
cg_update_p_kernel(typename Prec<R>::G* p, const typename Prec<R>::G* __restrict__ r, long long ngroups, int BS, int nrhs,
                   const double* __restrict__ rr_new, const double* __restrict__ rr_old) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int rhs = (int)((e / BS) % nrhs);
    const R beta = rr_old[rhs] != 0.0 ? (R)(rr_new[rhs] / rr_old[rhs]) : R(0);
    for (; e < ngroups; e += stride) {
        const CV<V> rv = unpack(ldg_nc(r + e));
        CV<V> pp = unpack(p[e]);
        pp.re = vfma(beta, pp.re, rv.re); pp.im = vfma(beta, pp.im, rv.im);
        p[e] = pack(pp);
    }
}

// ------------------------------------------------------------------------------------------------
// N4. BiCGSTAB vector updates (van der Vorst, PAPER.md ref. [31] L671; Table V), one right-hand side, full fields.
// All scalars live on the device in per-iteration slots of 8 doubles (dwf_bicgstab_pv in dwf_api.cu):
//   slot(i) = { rho_i (re, im), <rhat0, v_i> (re, im), <t_i, s_i> (re, im), <t_i, t_i>, |r_i|^2 },   rho_i = <rhat0, r_{i-1}>
//   alpha_i = rho_i / <rhat0, v_i>,  omega_i = <t_i, s_i> / <t_i, t_i>,  beta_i = (rho_i / rho_{i-1}) (alpha_{i-1} / omega_{i-1}).
// A zero denominator (zero or exactly converged right-hand side) freezes the iteration: the coefficient is 0.
// ------------------------------------------------------------------------------------------------
struct cd { double re, im; };
__device__ __forceinline__ cd cd_div(cd a, cd b) {
    const double n = b.re * b.re + b.im * b.im;
    if (n == 0.0) return {0.0, 0.0};
    return {(a.re * b.re + a.im * b.im) / n, (a.im * b.re - a.re * b.im) / n};
}
__device__ __forceinline__ cd cd_mul(cd a, cd b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ cd bicg_alpha(const double* slot) { return cd_div({slot[0], slot[1]}, {slot[2], slot[3]}); }
__device__ __forceinline__ cd bicg_omega(const double* slot) {
    return slot[6] != 0.0 ? cd{slot[4] / slot[6], slot[5] / slot[6]} : cd{0.0, 0.0};
}
// y += a x  for complex a, lane vectors
template <typename R, typename V> __device__ __forceinline__ void caxpy(CV<V>& y, R are, R aim, const CV<V>& x) {
    y.re = vfnma(aim, x.im, vfma(are, x.re, y.re));
    y.im = vfma(aim, x.re, vfma(are, x.im, y.im));
}

// Fixed-order combine of per-thread sums (4 components) into per-block partials partial[blockIdx.x * 4 + c]: a binary tree over
// the 256 threads in shared memory (deterministic).
__device__ __forceinline__ void block_combine4(double a0, double a1, double a2, double a3, double* partial) {
    __shared__ double s4[4][256];
    const int t = threadIdx.x;
    s4[0][t] = a0; s4[1][t] = a1; s4[2][t] = a2; s4[3][t] = a3;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (t < w) { s4[0][t] += s4[0][t + w]; s4[1][t] += s4[1][t + w]; s4[2][t] += s4[2][t + w]; s4[3][t] += s4[3][t + w]; }
        __syncthreads();
    }
    if (t < 4) partial[(size_t)blockIdx.x * 4 + t] = s4[t][0];
}
// out[c] = sum over blocks of partial[k*4 + c] for the components c with out_idx[c] >= 0 (written to out[out_idx[c]])
__global__ void __launch_bounds__(256)
reduce_final4_kernel(const double* __restrict__ partial, int nblocks, double* out, int i0, int i1, int i2, int i3) {
    __shared__ double s4[4][256];
    const int t = threadIdx.x;
    double a[4] = {0, 0, 0, 0};
    for (int k = t; k < nblocks; k += 256)
#pragma unroll
        for (int c = 0; c < 4; c++) a[c] += partial[(size_t)k * 4 + c];
#pragma unroll
    for (int c = 0; c < 4; c++) s4[c][t] = a[c];
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (t < w) {
#pragma unroll
            for (int c = 0; c < 4; c++) s4[c][t] += s4[c][t + w];
        }
        __syncthreads();
    }
    if (t == 0) {
        const int idx[4] = {i0, i1, i2, i3};
#pragma unroll
        for (int c = 0; c < 4; c++) if (idx[c] >= 0) out[idx[c]] = s4[c][0];
    }
}

// partials {Re<x,y>, Im<x,y>, <x,x>, 0}
template <typename R>
__global__ void __launch_bounds__(256)
inner_pair_kernel(const typename Prec<R>::G* __restrict__ x, const typename Prec<R>::G* __restrict__ y, long long ngroups, double* partial) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    double sre = 0, sim = 0, nre = 0, nim = 0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < ngroups; e += stride) {
        const CV<V> xx = unpack(ldg_nc(x + e)), yy = unpack(ldg_nc(y + e));
        acc_inner(sre, sim, xx, yy);
        acc_inner(nre, nim, xx, xx);
    }
    block_combine4(sre, sim, nre, 0.0, partial);
}

// init: r = b - q (q = A x_0), rhat0 = r, p = v = 0; partials {|r|^2, 0, |r|^2, 0} (rho_1 = <rhat0, r_0> = |r_0|^2)
template <typename R>
__global__ void __launch_bounds__(256)
bicg_init_kernel(const typename Prec<R>::G* __restrict__ b, const typename Prec<R>::G* __restrict__ q, typename Prec<R>::G* r,
                 typename Prec<R>::G* rhat, long long ngroups, double* partial) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    double sre = 0, sim = 0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < ngroups; e += stride) {
        const CV<V> rr = csub(unpack(ldg_nc(b + e)), unpack(ldg_nc(q + e)));
        r[e] = pack(rr); rhat[e] = pack(rr);
        acc_inner(sre, sim, rr, rr);
    }
    block_combine4(sre, 0.0, sre, 0.0, partial);
}

// p = r + beta (p - omega_{i-1} v);  first iteration: p = r
template <typename R>
__global__ void __launch_bounds__(256)
bicg_p_kernel(typename Prec<R>::G* p, const typename Prec<R>::G* __restrict__ r, const typename Prec<R>::G* __restrict__ v,
              long long ngroups, const double* __restrict__ slot_prev, const double* __restrict__ slot, int first) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    cd beta = {0, 0}, om = {0, 0};
    if (!first) {
        om = bicg_omega(slot_prev);
        beta = cd_mul(cd_div({slot[0], slot[1]}, {slot_prev[0], slot_prev[1]}), cd_div(bicg_alpha(slot_prev), om));
    }
    const R bre = (R)beta.re, bim = (R)beta.im, ore = (R)(-om.re), oim = (R)(-om.im);
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < ngroups; e += stride) {
        CV<V> out = unpack(ldg_nc(r + e));
        if (!first) {
            CV<V> d = unpack(p[e]);
            caxpy<R>(d, ore, oim, unpack(ldg_nc(v + e)));          // p - omega v
            caxpy<R>(out, bre, bim, d);
        }
        p[e] = pack(out);
    }
}

// s = r - alpha_i v   (in place: s overwrites r)
template <typename R>
__global__ void __launch_bounds__(256)
bicg_s_kernel(typename Prec<R>::G* r, const typename Prec<R>::G* __restrict__ v, long long ngroups, const double* __restrict__ slot) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const cd al = bicg_alpha(slot);
    const R are = (R)(-al.re), aim = (R)(-al.im);
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < ngroups; e += stride) {
        CV<V> s = unpack(r[e]);
        caxpy<R>(s, are, aim, unpack(ldg_nc(v + e)));
        r[e] = pack(s);
    }
}

// x += alpha_i p + omega_i s ;  r = s - omega_i t  (in place over s);  partials {|r|^2, 0, Re<rhat0, r>, Im<rhat0, r>}
template <typename R>
__global__ void __launch_bounds__(256)
bicg_xr_kernel(typename Prec<R>::G* x, typename Prec<R>::G* sr, const typename Prec<R>::G* __restrict__ p,
               const typename Prec<R>::G* __restrict__ t, const typename Prec<R>::G* __restrict__ rhat, long long ngroups,
               const double* __restrict__ slot, double* partial) {
    using V = typename Prec<R>::V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const cd al = bicg_alpha(slot), om = bicg_omega(slot);
    const R are = (R)al.re, aim = (R)al.im, ore = (R)om.re, oim = (R)om.im;
    double nre = 0, nim = 0, hre = 0, him = 0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < ngroups; e += stride) {
        CV<V> xx = unpack(x[e]);
        CV<V> s = unpack(sr[e]);
        caxpy<R>(xx, are, aim, unpack(ldg_nc(p + e)));
        caxpy<R>(xx, ore, oim, s);
        x[e] = pack(xx);
        caxpy<R>(s, (R)(-om.re), (R)(-om.im), unpack(ldg_nc(t + e)));
        sr[e] = pack(s);
        acc_inner(nre, nim, s, s);
        acc_inner(hre, him, unpack(ldg_nc(rhat + e)), s);
    }
    block_combine4(nre, 0.0, hre, him, partial);
}

}  // namespace dwf
