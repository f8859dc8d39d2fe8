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

#ifndef HOP_THREADS
#define HOP_THREADS 128       // threads per CTA of the stencil kernel (a CTA covers HOP_THREADS / K sites)
#endif

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
    int Ls, nrhs;          // runtime Ls (used when the kernel's LS template parameter is 0)
    int r0, rn;            // this launch covers right-hand sides r0 .. r0+rn-1
    int parity0;           // output parity of slot 0
    int nslots;            // 1: one output parity; 2: both, interleaved in chunks of chunk_groups site groups
    int GS;                // sites per CTA (a CTA = one group of G consecutive sites x one rhs x K lane groups)
    int sg_shift;          // log2 of the site-group size of the block order; 0 = [site][rhs]
    // tiled kernel only (dwf_tile.cuh):
    const R* glinks[2];    // [p] gathered links of parity-p sites: [site][mu][fwd 18 | bwd 18] x (-1/2), 16 B pad per site
    R sigma;               // res = sigma * hop' + self  with hop' built from the (-1/2)-scaled links
    R moo_kappa, moo_v0scale;   // fused M_oo^-1 epilogue: 1/(5-M5), kappa / (1 + m kappa^Ls)
    unsigned* dyn_counter; // tiled kernel, non-NORM variants: [0] items handed out beyond the first two rounds, [1] CTAs that left (NULL: static assignment)
    unsigned items_per_rhs; // tiled kernel: != 0: items are ordered rhs-major, this many per right-hand side (0: tile-major, rhs-minor)
    long long item0;       // this launch covers work items item0 .. nitems-1 (a partial launch covers whole lattice blocks)
    long long nitems;      // end of the work items (tile | site group, rhs, parity slot) of this launch
    double* norm_partial;  // NORM epilogue: |out|^2 partials [CTA][warp][2] (each warp's running sum over its items, in item order)
    double* norm_out;      // ... summed in (CTA, warp) order by the last CTA to finish and written here
    unsigned* ticket;      // ... CTA completion counter (zero on entry, reset to zero by the last CTA)
    const double* ax_num;  // AXPBY with a device scalar: if non-NULL, ax_a = -(*ax_num / *ax_den) (0 when *ax_den == 0):
    const double* ax_den;  //   the CG residual update r <- r - alpha q fused into the launch that produces q
    long long ngroups;     // ceil(V4h / G)
    long long chunk_groups;
    R c_hop, c_diag, mass;
    R ax_a, ax_b, ax_c;
    R g5_shift;            // G5 epilogue: res = Gamma5 (hop + self) + g5_shift * in   (H_DW + shift; 0: none)
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
// shared-memory link slot: 16-byte aligned, LINK_SLOT reals (fp32: 18 reals padded to 20; fp64: 18)
template <typename R> struct LinkSmem;
template <> struct LinkSmem<float>  { static constexpr int SLOT = 20; static constexpr int SITE = 8 * 20 + 4; };   // 656 B per site
template <> struct LinkSmem<double> { static constexpr int SLOT = 18; static constexpr int SITE = 8 * 18 + 2; };   // 1168 B per site

// core of one direction: project p (12 components) to a half spinor, multiply by the link u, reconstruct, accumulate
template <int MU, int SG, bool FWD, typename R, typename V>
__device__ __forceinline__ void hop_dir_core(CV<V> (&acc)[12], const CV<V> (&p)[12], const R (&u)[18]) {
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

template <int MU, int SG, bool FWD, typename R, typename V, typename G>
__device__ __forceinline__ void hop_dir(CV<V> (&acc)[12], const G* __restrict__ psi, const int cstride,
                                        const R* __restrict__ link /* shared memory */) {
    CV<V> p[12];
#pragma unroll
    for (int c = 0; c < 12; c++) p[c] = unpack(ldg_nc(psi + c * cstride));
    R u[18];
    if constexpr (sizeof(R) == 4) {
        const float4* l4 = reinterpret_cast<const float4*>(link);
#pragma unroll
        for (int k = 0; k < 4; k++) { float4 t = l4[k]; u[4 * k] = t.x; u[4 * k + 1] = t.y; u[4 * k + 2] = t.z; u[4 * k + 3] = t.w; }
        const float2 t2 = *reinterpret_cast<const float2*>(link + 16);
        u[16] = t2.x; u[17] = t2.y;
    } else {
        const double2* l2 = reinterpret_cast<const double2*>(link);
#pragma unroll
        for (int k = 0; k < 9; k++) { double2 t = l2[k]; u[2 * k] = t.x; u[2 * k + 1] = t.y; }
    }
    hop_dir_core<MU, SG, FWD>(acc, p, u);
}

// ---- the 4D-site-diagonal part of eq. 4: res[c] += c_diag psi(s) + coef psi(s -+ 1) ----------------
// Components c < 6 are the P_+ half (spins 0,1), c >= 6 the P_- half (R2).  Non-adjoint: P_+ couples
// to s-1 (wall: +m psi(Ls-1) at s = 0), P_- to s+1 (wall: +m psi(0) at s = Ls-1).  Adjoint: swapped.
//
// fp32: this thread holds lanes (sa, sb) = (2k, 2k+1) of its (site, rhs) block (K = Ls/2 groups per component).
//   "s-1" rule: neighbours (2k-1, 2k)   = (prev group .y, own .x), coefficients (k==0 ? m : -1, -1)
//   "s+1" rule: neighbours (2k+1, 2k+2) = (own .y, next group .x), coefficients (-1, k==last ? m : -1)
template <bool DAG>
__device__ __forceinline__ void self_term(CV<float2> (&res)[12], const float4* __restrict__ blk,
                                          const int K, const int k, float c_diag, float mass) {
    const int kprev = (k == 0) ? K - 1 : k - 1;
    const int knext = (k == K - 1) ? 0 : k + 1;
    const float2 coef_dn = make_float2((k == 0) ? mass : -1.f, -1.f);
    const float2 coef_up = make_float2(-1.f, (k == K - 1) ? mass : -1.f);
    const float4* own_p = blk + k;
    const float4* dn_p = blk + kprev;
    const float4* up_p = blk + knext;
    // When K divides 32 the K threads of a block sit in one warp: fetch the s-1 / s+1 lanes by shuffle.
    const bool shfl = (K == 4 || K == 8 || K == 16 || K == 32);
    const int lane = threadIdx.x & 31;
    const unsigned mask = __activemask();                    // whole K-groups leave together, sources stay in-group
    const int src_dn = lane - k + kprev, src_up = lane - k + knext;
#pragma unroll
    for (int c = 0; c < 12; c++) {
        const CV<float2> own = unpack(ldg_nc(own_p + c * K));
        const bool down = DAG ? (c >= 6) : (c < 6);          // couples to s-1 ?
        CV<float2> t; float2 coef;
        if (down) {
            float oy_re, oy_im;
            if (shfl) { oy_re = __shfl_sync(mask, own.re.y, src_dn); oy_im = __shfl_sync(mask, own.im.y, src_dn); }
            else { const CV<float2> o = unpack(ldg_nc(dn_p + c * K)); oy_re = o.re.y; oy_im = o.im.y; }
            t.re = make_float2(oy_re, own.re.x); t.im = make_float2(oy_im, own.im.x); coef = coef_dn;
        } else {
            float ox_re, ox_im;
            if (shfl) { ox_re = __shfl_sync(mask, own.re.x, src_up); ox_im = __shfl_sync(mask, own.im.x, src_up); }
            else { const CV<float2> o = unpack(ldg_nc(up_p + c * K)); ox_re = o.re.x; ox_im = o.im.x; }
            t.re = make_float2(own.re.y, ox_re); t.im = make_float2(own.im.y, ox_im); coef = coef_up;
        }
        // the shifted-lane terms as scalar FMAs: no re-packing of (s-1 | s) pairs into aligned register pairs (2 MOVs per pair)
        float2 rr = vfma(c_diag, own.re, res[c].re), ri = vfma(c_diag, own.im, res[c].im);
        rr.x = fmaf(coef.x, t.re.x, rr.x); rr.y = fmaf(coef.y, t.re.y, rr.y);
        ri.x = fmaf(coef.x, t.im.x, ri.x); ri.y = fmaf(coef.y, t.im.y, ri.y);
        res[c].re = rr; res[c].im = ri;
    }
}

// fp64: this thread holds lane s = k of its (site, rhs) block (K = Ls).
template <bool DAG>
__device__ __forceinline__ void self_term(CV<double> (&res)[12], const double2* __restrict__ blk,
                                          const int K, const int k, double c_diag, double mass) {
    const int sprev = (k == 0) ? K - 1 : k - 1;
    const int snext = (k == K - 1) ? 0 : k + 1;
    const double coef_dn = (k == 0) ? mass : -1.0;
    const double coef_up = (k == K - 1) ? mass : -1.0;
    // When K divides 32 the K threads of a block sit in one warp: fetch the s-1 / s+1 lane by shuffle.
    const bool shfl = (K == 4 || K == 8 || K == 16 || K == 32);
    const int lane = threadIdx.x & 31;
    const unsigned mask = __activemask();
    const int src_dn = lane - k + sprev, src_up = lane - k + snext;
#pragma unroll
    for (int c = 0; c < 12; c++) {
        const CV<double> own = unpack(ldg_nc(blk + c * K + k));
        const bool down = DAG ? (c >= 6) : (c < 6);
        CV<double> o;
        if (shfl) { o.re = __shfl_sync(mask, own.re, down ? src_dn : src_up); o.im = __shfl_sync(mask, own.im, down ? src_dn : src_up); }
        else o = unpack(ldg_nc(blk + c * K + (down ? sprev : snext)));
        const double coef = down ? coef_dn : coef_up;
        res[c].re = fma(coef, o.re, fma(c_diag, own.re, res[c].re));
        res[c].im = fma(coef, o.im, fma(c_diag, own.im, res[c].im));
    }
}

// Gamma5 = gamma5 R5 (eq. 6, R6): lane group k of a block goes to group K-1-k (fp32: the two lanes
// of the group also swap).
//
// Generic stencil kernel (any even lattice >= 4, any even Ls; the production path for lattices made of whole tiles is
// hop_tile_kernel in dwf_tile.cuh).  A CTA of HOP_THREADS threads handles min(HOP_THREADS/8, HOP_THREADS/K) consecutive
// sites for ONE right-hand side; thread = (site, lane group k).  The 8 links of each of the CTA's sites are fetched once
// per CTA into shared memory and read back as 128-bit broadcasts; neighbour blocks come through L1 (LDG.NC).
template <typename R, int LS, bool DAG, bool HOP, bool SELF, bool G5, bool AXPBY>
__global__ void __launch_bounds__(HOP_THREADS, 512 / HOP_THREADS)
hop_kernel(const HopArgs<R> a) {
    using V = typename Prec<R>::V;
    using G = typename Prec<R>::G;
    constexpr int VL = Prec<R>::VL;
    constexpr int SLOT = LinkSmem<R>::SLOT, SITE = LinkSmem<R>::SITE;
    const int K = (LS > 0) ? LS / VL : a.Ls / VL;            // lane groups per component of a (site, rhs) block
    __shared__ __align__(16) R s_link[HOP ? (HOP_THREADS / 8) * SITE : 4];

    // ---- which (output parity slot, site group, rhs) is this CTA? -------------------------------------
    const long long bid = a.item0 + blockIdx.x;
    long long gg = bid / a.rn;                                // site group, maybe across both slots
    const int r = a.r0 + (int)(bid - gg * a.rn);
    int pi = 0;
    if (a.nslots == 2) {                                      // chunks of chunk_groups alternate between the parities
        const long long q = gg / (2 * a.chunk_groups);
        const long long rem = gg - q * 2 * a.chunk_groups;
        pi = rem >= a.chunk_groups;
        gg = q * a.chunk_groups + (rem - pi * a.chunk_groups);
    }
    if (gg >= a.ngroups) return;                              // uniform over the CTA
    const int p = (a.parity0 + pi) & 1;
    const long long site0 = gg * a.GS;

    if constexpr (HOP) {                                      // cooperative link fetch: thread t -> (site t/8, direction t%8)
        const int ls = threadIdx.x >> 3, d = threadIdx.x & 7;
        const long long st = site0 + ls;
        if (ls < a.GS && st < a.V4h) {
            const R* src;
            if ((d & 1) == 0) src = a.gauge[p] + (size_t)st * 72 + (d >> 1) * 18;
            else { const int n = __ldg(a.nbr[pi] + st * 8 + d); src = a.gauge[p ^ 1] + (size_t)n * 72 + (d >> 1) * 18; }
            R* dst = s_link + ls * SITE + d * SLOT;
            if constexpr (sizeof(R) == 4) {
                const float2* s2 = reinterpret_cast<const float2*>(src);
                float2* d2 = reinterpret_cast<float2*>(dst);
#pragma unroll
                for (int j = 0; j < 9; j++) d2[j] = __ldg(s2 + j);
            } else {
                const double2* s2 = reinterpret_cast<const double2*>(src);
                double2* d2 = reinterpret_cast<double2*>(dst);
#pragma unroll
                for (int j = 0; j < 9; j++) d2[j] = __ldg(s2 + j);
            }
        }
        __syncthreads();
    }
    const int ls = threadIdx.x / K;                           // site within the tile
    const int k = threadIdx.x - ls * K;
    const long long site = site0 + ls;
    if (ls >= a.GS || site >= a.V4h) return;
    const int BS = 12 * K;                                    // groups per (site, rhs) block
    const long long blk = blk_index(site, r, a.nrhs, a.sg_shift);

    CV<V> acc[12];
#pragma unroll
    for (int c = 0; c < 12; c++) { acc[c].re = vzero(V()); acc[c].im = vzero(V()); }

    if constexpr (HOP) {
        const int4* nb4 = reinterpret_cast<const int4*>(a.nbr[pi] + site * 8);
        const int4 n0 = __ldg(nb4), n1 = __ldg(nb4 + 1);
        const G* in = a.in_hop[pi] + k;
        auto nb = [&](int n) -> const G* { return in + (size_t)blk_index(n, r, a.nrhs, a.sg_shift) * BS; };
        const R* u = s_link + ls * SITE;
        constexpr int SF = DAG ? +1 : -1;                     // projector sign on the forward hop
        hop_dir<0, SF, true >(acc, nb(n0.x), K, u + 0 * SLOT);
        hop_dir<0, -SF, false>(acc, nb(n0.y), K, u + 1 * SLOT);
        hop_dir<1, SF, true >(acc, nb(n0.z), K, u + 2 * SLOT);
        hop_dir<1, -SF, false>(acc, nb(n0.w), K, u + 3 * SLOT);
        hop_dir<2, SF, true >(acc, nb(n1.x), K, u + 4 * SLOT);
        hop_dir<2, -SF, false>(acc, nb(n1.y), K, u + 5 * SLOT);
        hop_dir<3, SF, true >(acc, nb(n1.z), K, u + 6 * SLOT);
        hop_dir<3, -SF, false>(acc, nb(n1.w), K, u + 7 * SLOT);
#pragma unroll
        for (int c = 0; c < 12; c++) { acc[c].re = vmul(a.c_hop, acc[c].re); acc[c].im = vmul(a.c_hop, acc[c].im); }
    }
    if constexpr (SELF) {
        self_term<DAG>(acc, a.in_self[pi] + (size_t)blk * BS, K, k, a.c_diag, a.mass);
    }
    int ko = k;
    if constexpr (G5) {
        ko = K - 1 - k;
#pragma unroll
        for (int c = 0; c < 12; c++) {
            acc[c].re = vswap(acc[c].re); acc[c].im = vswap(acc[c].im);
            if (c >= 6) { acc[c].re = vneg(acc[c].re); acc[c].im = vneg(acc[c].im); }
        }
        if (SELF && a.g5_shift != R(0)) {                     // res = (H_DW + shift) in, see dwf_tile.cuh
            const G* t = a.in_self[pi] + (size_t)blk * BS + ko;
#pragma unroll
            for (int c = 0; c < 12; c++) {
                const CV<V> tt = unpack(ldg_nc(t + c * K));
                acc[c].re = vfma(a.g5_shift, tt.re, acc[c].re); acc[c].im = vfma(a.g5_shift, tt.im, acc[c].im);
            }
        }
    }
    const size_t obase = (size_t)blk * BS + ko;
    if constexpr (AXPBY) {
        const G* y = a.y[pi] + obase;
        const G* z = a.z[pi] + obase;
#pragma unroll
        for (int c = 0; c < 12; c++) {
            const CV<V> yy = unpack(ldg_nc(y + c * K));
            const CV<V> zz = unpack(ld_plain(z + c * K));
            acc[c].re = vfma(a.ax_c, zz.re, vfma(a.ax_b, yy.re, vmul(a.ax_a, acc[c].re)));
            acc[c].im = vfma(a.ax_c, zz.im, vfma(a.ax_b, yy.im, vmul(a.ax_a, acc[c].im)));
        }
    }
    G* o = a.out[pi] + obase;
#pragma unroll
    for (int c = 0; c < 12; c++) o[c * K] = pack(acc[c]);
}

}  // namespace dwf
