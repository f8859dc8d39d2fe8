// dwf_hop.cuh -- the D_hop stencil kernel with fused D_DW / H_DW / Schur / Chebyshev epilogues.
//
// One kernel computes, for every output 4D site x of parity p and every lane group (fifth-dimension
// slices s and right-hand sides r):
//
//   hop(x,s)    = sum_mu (1 -+ gamma_mu) U_mu(x) in_hop(x+mu,s) + (1 +- gamma_mu) U_mu^dag(x-mu) in_hop(x-mu,s)
//                                                          PAPER.md eq. 2 L30 (upper sign; lower = adjoint)
//   self(x,s)   = (5-M5) in_self(x,s) - P_-+ in_self(x,s+1) - P_+- in_self(x,s-1)  (+ m walls)
//                                                          eq. 4 L39 / eq. 5: the 4D-site-diagonal part
//   res         = c_hop * hop + self                       D_DW: c_hop = -1/2 ; Schur K2: c_hop = -1/4
//   res         = Gamma5 res = gamma5 res(x, Ls-1-s)       eq. 6 L48 (H_DW), optional
//   out         = a res + b Y + c Z                        Chebyshev three-term recurrence, optional
//
// The spin projection to half spinors happens before the SU(3) multiply (12 instead of 24 complex
// multiplies-by-a-link per direction); the antiperiodic-t sign lives in the stored links.
#pragma once
#include "dwf_vec.cuh"

namespace dwf {

template <typename R> struct HopArgs {
    using G = typename Prec<R>::G;
    const G* in_hop[2];    // [p] half field of parity 1-p that feeds output parity p
    const G* in_self[2];   // [p] half field of parity p (self term)
    G* out[2];             // [p]
    const G* y[2];         // [p] axpby operands, located like the output
    const G* z[2];         //     (z may alias out: each thread reads its location before writing it)
    const R* gauge[2];     // [q] links stored at sites of parity q: [V4h][mu 4][18 reals]
    const int* nbr[2];     // [p] neighbour table of parity-p sites: [V4h][8], slot 2mu = +mu, 2mu+1 = -mu
    long long V4h;
    int Ls, nrhs, NLG;     // NLG = nrhs * Ls / VL lane groups per site
    int parity0;           // output parity of blockIdx.y == 0
    R c_hop, c_diag, mass;
    R ax_a, ax_b, ax_c;
};

// (U h)_a = sum_b U_ab h_b  (FWD)   or   (U^dag h)_a = sum_b conj(U_ba) h_b  (!FWD)
template <bool FWD, typename R, typename V>
__device__ __forceinline__ void su3_mul(const R (&u)[18], const CV<V> (&h)[3], CV<V> (&g)[3]) {
#pragma unroll
    for (int a = 0; a < 3; a++) {
        V re, im;
#pragma unroll
        for (int b = 0; b < 3; b++) {
            const R ur = FWD ? u[(a * 3 + b) * 2] : u[(b * 3 + a) * 2];
            const R ui = FWD ? u[(a * 3 + b) * 2 + 1] : u[(b * 3 + a) * 2 + 1];
            if (b == 0) { re = vmul(ur, h[0].re); im = vmul(ur, h[0].im); }
            else        { re = vfma(ur, h[b].re, re); im = vfma(ur, h[b].im, im); }
            if (FWD) { re = vfnma(ui, h[b].im, re); im = vfma(ui, h[b].re, im); }
            else     { re = vfma(ui, h[b].im, re);  im = vfnma(ui, h[b].re, im); }
        }
        g[a].re = re; g[a].im = im;
    }
}

// One direction of the stencil.  MU = 0..3 (x,y,z,t); SG = -1: projector (1 - gamma_mu), +1: (1 + gamma_mu)
// (chiral basis R1; the rank-2 forms below are the rows of the 4x4 matrices written out).
template <int MU, int SG, bool FWD, typename R, typename V, typename G>
__device__ __forceinline__ void hop_dir(CV<V> (&acc)[12], const G* __restrict__ psi, size_t cstride,
                                        const R* __restrict__ link) {
    CV<V> p[12];
#pragma unroll
    for (int c = 0; c < 12; c++) p[c] = unpack(ldg_nc(psi + c * cstride));
    R u[18];
    if constexpr (sizeof(R) == 4) {
        const float2* l2 = reinterpret_cast<const float2*>(link);
#pragma unroll
        for (int k = 0; k < 9; k++) { float2 t = __ldg(l2 + k); u[2 * k] = t.x; u[2 * k + 1] = t.y; }
    } else {
        const double2* l2 = reinterpret_cast<const double2*>(link);
#pragma unroll
        for (int k = 0; k < 9; k++) { double2 t = __ldg(l2 + k); u[2 * k] = t.x; u[2 * k + 1] = t.y; }
    }
    CV<V> h0[3], h1[3], g0[3], g1[3];
#pragma unroll
    for (int col = 0; col < 3; col++) {
        const CV<V> p0 = p[col], p1 = p[3 + col], p2 = p[6 + col], p3 = p[9 + col];
        if constexpr (MU == 0) {
            if constexpr (SG < 0) { h0[col] = caddi(p0, p3); h1[col] = caddi(p1, p2); }
            else                  { h0[col] = csubi(p0, p3); h1[col] = csubi(p1, p2); }
        } else if constexpr (MU == 1) {
            if constexpr (SG < 0) { h0[col] = cadd(p0, p3); h1[col] = csub(p1, p2); }
            else                  { h0[col] = csub(p0, p3); h1[col] = cadd(p1, p2); }
        } else if constexpr (MU == 2) {
            if constexpr (SG < 0) { h0[col] = caddi(p0, p2); h1[col] = csubi(p1, p3); }
            else                  { h0[col] = csubi(p0, p2); h1[col] = caddi(p1, p3); }
        } else {
            if constexpr (SG < 0) { h0[col] = csub(p0, p2); h1[col] = csub(p1, p3); }
            else                  { h0[col] = cadd(p0, p2); h1[col] = cadd(p1, p3); }
        }
    }
    su3_mul<FWD>(u, h0, g0);
    su3_mul<FWD>(u, h1, g1);
#pragma unroll
    for (int col = 0; col < 3; col++) {
        acc[col] = cadd(acc[col], g0[col]);
        acc[3 + col] = cadd(acc[3 + col], g1[col]);
        if constexpr (MU == 0) {
            if constexpr (SG < 0) { acc[6 + col] = csubi(acc[6 + col], g1[col]); acc[9 + col] = csubi(acc[9 + col], g0[col]); }
            else                  { acc[6 + col] = caddi(acc[6 + col], g1[col]); acc[9 + col] = caddi(acc[9 + col], g0[col]); }
        } else if constexpr (MU == 1) {
            if constexpr (SG < 0) { acc[6 + col] = csub(acc[6 + col], g1[col]); acc[9 + col] = cadd(acc[9 + col], g0[col]); }
            else                  { acc[6 + col] = cadd(acc[6 + col], g1[col]); acc[9 + col] = csub(acc[9 + col], g0[col]); }
        } else if constexpr (MU == 2) {
            if constexpr (SG < 0) { acc[6 + col] = csubi(acc[6 + col], g0[col]); acc[9 + col] = caddi(acc[9 + col], g1[col]); }
            else                  { acc[6 + col] = caddi(acc[6 + col], g0[col]); acc[9 + col] = csubi(acc[9 + col], g1[col]); }
        } else {
            if constexpr (SG < 0) { acc[6 + col] = csub(acc[6 + col], g0[col]); acc[9 + col] = csub(acc[9 + col], g1[col]); }
            else                  { acc[6 + col] = cadd(acc[6 + col], g0[col]); acc[9 + col] = cadd(acc[9 + col], g1[col]); }
        }
    }
}

// ---- the 4D-site-diagonal part of eq. 4: res[c] += c_diag psi(s) + coef psi(s -+ 1) ----------------
// Components c < 6 are the P_+ half (spins 0,1), c >= 6 the P_- half (R2).  Non-adjoint: P_+ couples
// to s-1 (wall: +m psi(Ls-1) at s = 0), P_- to s+1 (wall: +m psi(0) at s = Ls-1).  Adjoint: swapped.
//
// fp32: this thread holds lanes (sa, sb) = (2k, 2k+1) of rhs r.
//   "s-1" rule: neighbours (2k-1, 2k)   = (prev group .y, own .x), coefficients (k==0 ? m : -1, -1)
//   "s+1" rule: neighbours (2k+1, 2k+2) = (own .y, next group .x), coefficients (-1, k==last ? m : -1)
template <bool DAG>
__device__ __forceinline__ void self_term(CV<float2> (&res)[12], const float4* __restrict__ site_base,
                                          size_t cstride, int lg, int Ls, float c_diag, float mass) {
    const int half = Ls >> 1;
    const int k = lg % half;
    const int r0 = lg - k;                                   // first group of this rhs
    const int kprev = (k == 0) ? half - 1 : k - 1;
    const int knext = (k == half - 1) ? 0 : k + 1;
    const float2 coef_dn = make_float2((k == 0) ? mass : -1.f, -1.f);
    const float2 coef_up = make_float2(-1.f, (k == half - 1) ? mass : -1.f);
#pragma unroll
    for (int c = 0; c < 12; c++) {
        const CV<float2> own = unpack(ldg_nc(site_base + c * cstride + lg));
        const bool down = DAG ? (c >= 6) : (c < 6);          // couples to s-1 ?
        CV<float2> t; float2 coef;
        if (down) {
            const CV<float2> o = unpack(ldg_nc(site_base + c * cstride + r0 + kprev));
            t.re = make_float2(o.re.y, own.re.x); t.im = make_float2(o.im.y, own.im.x); coef = coef_dn;
        } else {
            const CV<float2> o = unpack(ldg_nc(site_base + c * cstride + r0 + knext));
            t.re = make_float2(own.re.y, o.re.x); t.im = make_float2(own.im.y, o.im.x); coef = coef_up;
        }
        res[c].re = vfma2(coef, t.re, vfma(c_diag, own.re, res[c].re));
        res[c].im = vfma2(coef, t.im, vfma(c_diag, own.im, res[c].im));
    }
}

// fp64: this thread holds lane s of rhs r.
template <bool DAG>
__device__ __forceinline__ void self_term(CV<double> (&res)[12], const double2* __restrict__ site_base,
                                          size_t cstride, int lg, int Ls, double c_diag, double mass) {
    const int s = lg % Ls;
    const int r0 = lg - s;
    const int sprev = (s == 0) ? Ls - 1 : s - 1;
    const int snext = (s == Ls - 1) ? 0 : s + 1;
    const double coef_dn = (s == 0) ? mass : -1.0;
    const double coef_up = (s == Ls - 1) ? mass : -1.0;
#pragma unroll
    for (int c = 0; c < 12; c++) {
        const CV<double> own = unpack(ldg_nc(site_base + c * cstride + lg));
        const bool down = DAG ? (c >= 6) : (c < 6);
        const CV<double> o = unpack(ldg_nc(site_base + c * cstride + r0 + (down ? sprev : snext)));
        const double coef = down ? coef_dn : coef_up;
        res[c].re = fma(coef, o.re, fma(c_diag, own.re, res[c].re));
        res[c].im = fma(coef, o.im, fma(c_diag, own.im, res[c].im));
    }
}

// Gamma5 = gamma5 R5 target lane group and lane swap (eq. 6, R6)
__device__ __forceinline__ int g5_target(int lg, int Ls, float) {
    const int half = Ls >> 1; const int k = lg % half; return lg - k + (half - 1 - k);
}
__device__ __forceinline__ int g5_target(int lg, int Ls, double) {
    const int s = lg % Ls; return lg - s + (Ls - 1 - s);
}

template <typename R, bool DAG, bool HOP, bool SELF, bool G5, bool AXPBY>
__global__ void __launch_bounds__(128)
hop_kernel(const HopArgs<R> a) {
    using V = typename Prec<R>::V;
    using G = typename Prec<R>::G;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long site = gid / a.NLG;
    if (site >= a.V4h) return;
    const int lg = (int)(gid - site * a.NLG);
    const int pi = blockIdx.y;                      // which output-parity slot
    const size_t cstride = (size_t)a.NLG;

    CV<V> acc[12];
#pragma unroll
    for (int c = 0; c < 12; c++) { acc[c].re = vzero(V()); acc[c].im = vzero(V()); }

    if constexpr (HOP) {
        const int p = (a.parity0 + pi) & 1;
        const int4* nb4 = reinterpret_cast<const int4*>(a.nbr[pi] + site * 8);
        const int4 n0 = __ldg(nb4), n1 = __ldg(nb4 + 1);
        const G* in = a.in_hop[pi] + lg;
        const R* u_own = a.gauge[p] + (size_t)site * 72;
        const R* u_nbr = a.gauge[p ^ 1];
        constexpr int SF = DAG ? +1 : -1;           // projector sign on the forward hop
        hop_dir<0, SF, true >(acc, in + (size_t)n0.x * 12 * cstride, cstride, u_own + 0);
        hop_dir<0, -SF, false>(acc, in + (size_t)n0.y * 12 * cstride, cstride, u_nbr + (size_t)n0.y * 72 + 0);
        hop_dir<1, SF, true >(acc, in + (size_t)n0.z * 12 * cstride, cstride, u_own + 18);
        hop_dir<1, -SF, false>(acc, in + (size_t)n0.w * 12 * cstride, cstride, u_nbr + (size_t)n0.w * 72 + 18);
        hop_dir<2, SF, true >(acc, in + (size_t)n1.x * 12 * cstride, cstride, u_own + 36);
        hop_dir<2, -SF, false>(acc, in + (size_t)n1.y * 12 * cstride, cstride, u_nbr + (size_t)n1.y * 72 + 36);
        hop_dir<3, SF, true >(acc, in + (size_t)n1.z * 12 * cstride, cstride, u_own + 54);
        hop_dir<3, -SF, false>(acc, in + (size_t)n1.w * 12 * cstride, cstride, u_nbr + (size_t)n1.w * 72 + 54);
#pragma unroll
        for (int c = 0; c < 12; c++) { acc[c].re = vmul(a.c_hop, acc[c].re); acc[c].im = vmul(a.c_hop, acc[c].im); }
    }
    if constexpr (SELF) {
        self_term<DAG>(acc, a.in_self[pi] + (size_t)site * 12 * cstride, cstride, lg, a.Ls, a.c_diag, a.mass);
    }
    int lgo = lg;
    if constexpr (G5) {
        lgo = g5_target(lg, a.Ls, R());
#pragma unroll
        for (int c = 0; c < 12; c++) {
            acc[c].re = vswap(acc[c].re); acc[c].im = vswap(acc[c].im);
            if (c >= 6) { acc[c].re = vneg(acc[c].re); acc[c].im = vneg(acc[c].im); }
        }
    }
    const size_t obase = (size_t)site * 12 * cstride + lgo;
    if constexpr (AXPBY) {
        const G* y = a.y[pi] + obase;
        const G* z = a.z[pi] + obase;
#pragma unroll
        for (int c = 0; c < 12; c++) {
            const CV<V> yy = unpack(ldg_nc(y + c * cstride));
            const CV<V> zz = unpack(ld_plain(z + c * cstride));
            acc[c].re = vfma(a.ax_c, zz.re, vfma(a.ax_b, yy.re, vmul(a.ax_a, acc[c].re)));
            acc[c].im = vfma(a.ax_c, zz.im, vfma(a.ax_b, yy.im, vmul(a.ax_a, acc[c].im)));
        }
    }
    G* o = a.out[pi] + obase;
#pragma unroll
    for (int c = 0; c < 12; c++) o[c * cstride] = pack(acc[c]);
}

}  // namespace dwf
