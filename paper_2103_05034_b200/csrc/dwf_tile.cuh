// dwf_tile.cuh -- the tiled, persistent form of the stencil kernel (same arithmetic as dwf_hop.cuh).
//
// Used when the lattice is made of whole tiles of TS sites per parity (TS = 32: 4x4x2x2, TS = 16:
// 4x2x2x2) and Ls is a compile-time size.  A work item is (tile, right-hand side, output parity);
// thread = (site in tile, lane group k); persistent CTAs walk the items in launch order.
//
// Everything a tile needs that is reused or needs an index lookup arrives in shared memory by bulk
// asynchronous copies (cp.async.bulk + mbarrier, SASS UBLKCP) issued one item ahead:
//   * the tile's TS opposite-parity sites ("interior": the only spinor blocks used by more than one
//     output site of the tile; one contiguous run of TS*BS groups thanks to the block order),
//   * the tile's gathered links  [site][mu][U_mu(x) | U_mu(x-mu)]  pre-scaled by -1/2 (set_gauge),
//   * the tile's neighbour table [site][8].
// Halo blocks (each used by exactly one output site) and the self / axpby operands are read from
// global memory.  res = sigma * hop' + self with hop' built from the scaled links (sigma = 1 for
// D_DW, H_DW, D_PV: no scaling pass).  The self term is computed first, while the copies land.
#pragma once
#include <type_traits>

#include "dwf_aux.cuh"
#include "dwf_hop.cuh"

#ifndef DWF_INT_STAGES
#define DWF_INT_STAGES 1     // shared-memory buffers for the tile interior (2: warps may run one item ahead)
#endif
#ifndef DWF_MINCTAS128
#define DWF_MINCTAS128 4
#endif
#ifndef DWF_MINCTAS192
#define DWF_MINCTAS192 2
#endif
#ifndef DWF_MINCTAS256
#define DWF_MINCTAS256 2
#endif

namespace dwf {

// ---- mbarrier + bulk async copy (TMA, 1-D) --------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    unsigned ok = 0;
    while (!ok)
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
}
// global -> shared bulk copy, completion signalled on the mbarrier (bytes: multiple of 16, 16-byte aligned)
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// gathered links of one site: 4 x (fwd 18 | bwd 18) reals + 16 bytes of padding, so that the four
// sites of a warp read distinct banks (592 B fp32, 1168 B fp64)
template <typename R> struct TileLinks { static constexpr int SITE = 4 * 36 + 16 / (int)sizeof(R); };

template <typename R, int LS, int TS> struct TileGeom {
    static constexpr int K = LS / Prec<R>::VL;
    static constexpr int THREADS = TS * K;
    static constexpr int MIN_CTAS = THREADS <= 128 ? DWF_MINCTAS128 : THREADS <= 192 ? DWF_MINCTAS192 : THREADS <= 256 ? DWF_MINCTAS256 : 1;
    static constexpr int BS = 12 * K;
    static constexpr unsigned INTERIOR_BYTES = TS * BS * 16;
    static constexpr unsigned LINK_BYTES = TS * TileLinks<R>::SITE * sizeof(R);
    static constexpr unsigned NBR_BYTES = TS * 8 * sizeof(int);
    static constexpr unsigned SMALL_BYTES = LINK_BYTES + NBR_BYTES;
    // the fused M_oo^-1 epilogue transposes the tile through the interior buffer with rows padded by one group
    static constexpr unsigned TRANS_BYTES = TS * 12 * (K + 1) * 16;
    static constexpr unsigned INT_STRIDE = INTERIOR_BYTES > TRANS_BYTES ? INTERIOR_BYTES : TRANS_BYTES;
    // Interior buffers: one.  With two CTAs per SM the refill of one CTA's buffer is covered by the other CTA; for the CTA that
    // has the SM to itself (384 threads: fp32 Ls 24) a second buffer was measured SLOWER on B200 (48^3x96x24 D_DW 28.3 ms
    // against 21.0 ms): the 72 KB it takes away from L1 cost more (halo and s+-1 loads hit L1) than the exposed refill.
    static constexpr int NSTI = DWF_INT_STAGES;
    static constexpr unsigned HDR = 256;     // mbarriers, counters, the queue of decoded work items
    static constexpr unsigned SMEM_BYTES = HDR + NSTI * INT_STRIDE + 2 * SMALL_BYTES;
};

// load the 18 reals of one link from the gathered shared-memory layout; HALF = 0: U_mu(x), 1: U_mu(x-mu)
template <int HALF>
__device__ __forceinline__ void load_link(const float* pair, float (&u)[18]) {
    if constexpr (HALF == 0) {
        const float4* l4 = reinterpret_cast<const float4*>(pair);
#pragma unroll
        for (int j = 0; j < 4; j++) { const float4 t = l4[j]; u[4 * j] = t.x; u[4 * j + 1] = t.y; u[4 * j + 2] = t.z; u[4 * j + 3] = t.w; }
        const float2 t2 = *reinterpret_cast<const float2*>(pair + 16);
        u[16] = t2.x; u[17] = t2.y;
    } else {                                                   // reals 18..35: 8-byte aligned head, then 16-byte aligned
        const float2 t2 = *reinterpret_cast<const float2*>(pair + 18);
        u[0] = t2.x; u[1] = t2.y;
        const float4* l4 = reinterpret_cast<const float4*>(pair + 20);
#pragma unroll
        for (int j = 0; j < 4; j++) { const float4 t = l4[j]; u[2 + 4 * j] = t.x; u[3 + 4 * j] = t.y; u[4 + 4 * j] = t.z; u[5 + 4 * j] = t.w; }
    }
}
template <int HALF>
__device__ __forceinline__ void load_link(const double* pair, double (&u)[18]) {
    const double2* l2 = reinterpret_cast<const double2*>(pair + 18 * HALF);
#pragma unroll
    for (int j = 0; j < 9; j++) { const double2 t = l2[j]; u[2 * j] = t.x; u[2 * j + 1] = t.y; }
}

// one direction: psi is a generic pointer (shared-memory interior block or global halo block)
template <int MU, int SG, bool FWD, typename R, typename V, typename G>
__device__ __forceinline__ void tile_dir(CV<V> (&acc)[12], const G* psi, const int cstride, const R* pair) {
    CV<V> p[12];
#pragma unroll
    for (int c = 0; c < 12; c++) p[c] = unpack(ld_plain(psi + c * cstride));
    R u[18];
    load_link<FWD ? 0 : 1>(pair, u);
    hop_dir_core<MU, SG, FWD>(acc, p, u);
}

template <typename R, int LS, int TS, bool DAG, bool HOP, bool SELF, bool G5, bool AXPBY, bool MOO = false, bool NORM = false>
__global__ void __launch_bounds__(TileGeom<R, LS, TS>::THREADS, TileGeom<R, LS, TS>::MIN_CTAS)
hop_tile_kernel(const HopArgs<R> a) {
    static_assert(!MOO || (HOP && !SELF && !G5 && !AXPBY), "fused M_oo^-1 follows a bare hop");
    using V = typename Prec<R>::V;
    using G = typename Prec<R>::G;
    using TG = TileGeom<R, LS, TS>;
    constexpr int K = TG::K, BS = TG::BS;
    constexpr int SH = (TS == 64) ? 6 : (TS == 32) ? 5 : 4;
    constexpr int LSITE = TileLinks<R>::SITE;
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int NSTI = TG::NSTI;
    unsigned long long* bar_int = reinterpret_cast<unsigned long long*>(smem);          // [NSTI]: interior landed
    unsigned long long* bar_small = reinterpret_cast<unsigned long long*>(smem) + 2;    // [2]: links + nbr landed
    unsigned char* s_small = smem + TG::HDR + NSTI * TG::INT_STRIDE;

    // work item w -> (tile gg, rhs r, parity slot pi): same order as the CTAs of the generic kernel
    const unsigned rn = (unsigned)a.rn, cg = (unsigned)a.chunk_groups;     // item counts fit 32 bits (checked by the host)
    auto decode = [&](long long w, long long& gg_out, int& r, int& pi) {
        unsigned gg;
        if (a.items_per_rhs) {                                 // rhs-major: all items of one right-hand side, then the next (one launch for the batch)
            const unsigned ri = (unsigned)w / a.items_per_rhs;
            gg = (unsigned)w - ri * a.items_per_rhs; r = a.r0 + (int)ri;
        } else {
            gg = (unsigned)w / rn;
            r = a.r0 + (int)((unsigned)w - gg * rn);
        }
        pi = 0;
        if (a.nslots == 2) {
            const unsigned q = gg / (2 * cg);
            const unsigned rem = gg - q * 2 * cg;
            pi = rem >= cg;
            gg = q * cg + (rem - pi * cg);
        }
        gg_out = gg;
    };
    auto issue_small_d = [&](long long gg, int pi, int buf) {  // one thread only
        const int p = (a.parity0 + pi) & 1;
        unsigned char* dst = s_small + buf * TG::SMALL_BYTES;
        mbar_expect_tx(bar_small + buf, TG::SMALL_BYTES);
        bulk_g2s(dst, a.glinks[p] + (size_t)gg * TS * LSITE, TG::LINK_BYTES, bar_small + buf);
        bulk_g2s(dst + TG::LINK_BYTES, a.nbr[pi] + (size_t)gg * TS * 8, TG::NBR_BYTES, bar_small + buf);
    };
    auto issue_interior_d = [&](long long gg, int r, int pi, int ib) {   // one thread only
        mbar_expect_tx(bar_int + ib, TG::INTERIOR_BYTES);
        bulk_g2s(smem + TG::HDR + ib * TG::INT_STRIDE, a.in_hop[pi] + (size_t)blk_index(gg * TS, r, a.nrhs, SH) * BS, TG::INTERIOR_BYTES, bar_int + ib);
    };
    auto issue_small = [&](long long w, int buf) { long long gg; int r, pi; decode(w, gg, r, pi); issue_small_d(gg, pi, buf); };
    auto issue_interior = [&](long long w, int ib) { long long gg; int r, pi; decode(w, gg, r, pi); issue_interior_d(gg, r, pi, ib); };

    // Which items does this CTA work on?  The first two are static (item0 + blockIdx.x, + gridDim.x), every further one is taken
    // from a global counter when the CTA gets there, two items ahead of its use (DYN).  Fast CTAs then take more items and the
    // items in flight stay one contiguous window of the sweep; with a static round-robin assignment the CTAs drift apart over the
    // rounds of a launch and the window -- the L2 footprint -- widens.  No result depends on who computes an item: the NORM
    // epilogue keeps one partial per (item, warp), summed in index order.
    constexpr bool DYN = (NSTI == 1);
    // the queue: slot it & 3 holds the decoded item of this CTA's sequence number it, {item, tile, rhs, parity slot}; item = nitems: none.
    // Only the refilling thread decodes (two integer divisions); the other threads read the slot.
    volatile int4* q_slot = reinterpret_cast<volatile int4*>(smem + 128);          // [4]
    volatile int* q_seq = reinterpret_cast<volatile int*>(smem + 112);             // highest sequence number whose slot is filled
    auto q_put = [&](int seq, long long w) -> bool {           // one thread only; returns whether there is such an item
        int4 v = make_int4((int)a.nitems, 0, 0, 0);
        if (w < a.nitems) { long long gg; int r, pi; decode(w, gg, r, pi); v = make_int4((int)w, (int)gg, r, pi); }
        q_slot[seq & 3].x = v.x; q_slot[seq & 3].y = v.y; q_slot[seq & 3].z = v.z; q_slot[seq & 3].w = v.w;
        return w < a.nitems;
    };
    const bool dyn = DYN && a.dyn_counter != nullptr;
    long long w = a.item0 + blockIdx.x;
    if (w >= a.nitems) return;                                 // the host never launches more CTAs than items
    unsigned* done_count = reinterpret_cast<unsigned*>(smem + 64);  // [2]: warps that finished the hop phase of even / odd items
    if (threadIdx.x == 0) {
        mbar_init(bar_int, 1); mbar_init(bar_int + 1, 1); mbar_init(bar_small, 1); mbar_init(bar_small + 1, 1);
        mbar_fence_init();
        done_count[0] = 0; done_count[1] = 0;
        { long long gg; int r, pi; decode(w, gg, r, pi);       // decode once, copies first
          issue_small_d(gg, pi, 0); issue_interior_d(gg, r, pi, 0);
          q_slot[0].x = (int)w; q_slot[0].y = (int)gg; q_slot[0].z = r; q_slot[0].w = pi; }
        if (q_put(1, w + gridDim.x)) { issue_small_d(q_slot[1].y, q_slot[1].w, 1); if (NSTI == 2) issue_interior_d(q_slot[1].y, q_slot[1].z, q_slot[1].w, 1); }
        *q_seq = 1;
    }
    __syncthreads();
    constexpr unsigned NWARPS = TG::THREADS / 32;

    const int ls = threadIdx.x / K;                            // site within the tile
    const int k = threadIdx.x - ls * K;

    R ax_a = a.ax_a;
    if constexpr (AXPBY) {
        if (a.ax_num) { const double den = *a.ax_den; ax_a = den != 0.0 ? (R)(-(*a.ax_num / den)) : R(0); }
    }
    for (int it = 0; ; it++) {
        long long gg; int r, pi;
        if constexpr (DYN) {
            while (*q_seq < it) __nanosleep(20);
            const volatile int4* sl = q_slot + (it & 3);
            w = sl->x; gg = sl->y; r = sl->z; pi = sl->w;
            if (w >= a.nitems) break;
        } else {
            if (it > 0) w += gridDim.x;
            if (w >= a.nitems) break;
            decode(w, gg, r, pi);
        }
        const long long wn = w + gridDim.x;                    // static assignment only
        const int buf = it & 1;
        const long long site = gg * TS + ls;
        const long long blk = blk_index(site, r, a.nrhs, SH);

        CV<V> acc[12];
#pragma unroll
        for (int c = 0; c < 12; c++) { acc[c].re = vzero(V()); acc[c].im = vzero(V()); }
        const bool scaled = (a.sigma != R(1));
        if constexpr (SELF) {                                  // global loads only: overlaps the copies in flight
            self_term<DAG>(acc, a.in_self[pi] + (size_t)blk * BS, K, k, a.c_diag, a.mass);
            if (HOP && scaled) {
                const R inv = R(1) / a.sigma;
#pragma unroll
                for (int c = 0; c < 12; c++) { acc[c].re = vmul(inv, acc[c].re); acc[c].im = vmul(inv, acc[c].im); }
            }
        }
        if constexpr (HOP) {
            mbar_wait(bar_small + buf, (it >> 1) & 1);
            const unsigned char* small = s_small + buf * TG::SMALL_BYTES;
            const int4* nb4 = reinterpret_cast<const int4*>(small + TG::LINK_BYTES) + ls * 2;
            const int4 n0 = nb4[0], n1 = nb4[1];
            const R* u = reinterpret_cast<const R*>(small) + ls * LSITE;
            const int ib = (NSTI == 2) ? buf : 0;
            const G* s_in = reinterpret_cast<const G*>(smem + TG::HDR + ib * TG::INT_STRIDE);
            const G* in = a.in_hop[pi] + k;
            // neighbour block: inside the tile -> shared memory, else global memory
            // blk_index(n, r) = n + (n >> SH) * (nrhs - 1) * TS + r * TS in 32 bits (launch_hop_t checks V4h * nrhs < 2^31): the 64-bit
            // form cost ~30 integer instructions per direction and thread
            const unsigned nb_c1 = (unsigned)(a.nrhs - 1) << SH, nb_c2 = (unsigned)r << SH;
            auto nb = [&](int n) -> const G* {
                const unsigned tn = (unsigned)n >> SH;
                if (tn == (unsigned)gg) return s_in + ((unsigned)n & (TS - 1)) * BS + k;
                return in + (size_t)((unsigned)n + tn * nb_c1 + nb_c2) * BS;
            };
            const G* q0 = nb(n0.x); const G* q1 = nb(n0.y); const G* q2 = nb(n0.z); const G* q3 = nb(n0.w);
            const G* q4 = nb(n1.x); const G* q5 = nb(n1.y); const G* q6 = nb(n1.z); const G* q7 = nb(n1.w);
            constexpr int SF = DAG ? +1 : -1;                  // projector sign on the forward hop
            mbar_wait(bar_int + ib, (NSTI == 2) ? (it >> 1) & 1 : it & 1);
            tile_dir<0, SF, true >(acc, q0, K, u + 0 * 36);
            tile_dir<0, -SF, false>(acc, q1, K, u + 0 * 36);
            tile_dir<1, SF, true >(acc, q2, K, u + 1 * 36);
            tile_dir<1, -SF, false>(acc, q3, K, u + 1 * 36);
            tile_dir<2, SF, true >(acc, q4, K, u + 2 * 36);
            tile_dir<2, -SF, false>(acc, q5, K, u + 2 * 36);
            tile_dir<3, SF, true >(acc, q6, K, u + 3 * 36);
            tile_dir<3, -SF, false>(acc, q7, K, u + 3 * 36);
            // The last warp to finish with the shared-memory buffers of this item refills them: the interior with
            // item it+1, this small buffer with item it+2 (nobody waits: arrival is awaited through the mbarriers).
            auto release_buffers = [&]() {
                __syncwarp();
                if ((threadIdx.x & 31) == 0) {
                    __threadfence_block();                     // this warp's reads of the buffers are performed before it counts itself done
                    const unsigned prev = atomicAdd(done_count + buf, 1u);
                    if (prev == (unsigned)((it >> 1) + 1) * NWARPS - 1) {
                        // generic-proxy accesses of the buffers (reads; the MOO transpose also writes) before the async-proxy refill
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        if constexpr (DYN) {
                            const volatile int4* s1 = q_slot + ((it + 1) & 3);     // filled one refill ago (or at the start)
                            const bool have1 = s1->x < (int)a.nitems;
                            if (have1) issue_interior_d(s1->y, s1->z, s1->w, 0);
                            long long w2 = a.nitems;
                            if (have1) w2 = dyn ? a.item0 + 2LL * gridDim.x + atomicAdd(a.dyn_counter, 1u) : (long long)s1->x + gridDim.x;
                            const bool have2 = q_put(it + 2, w2);
                            __threadfence_block();
                            *q_seq = it + 2;
                            if (have2) { const volatile int4* s2 = q_slot + ((it + 2) & 3); issue_small_d(s2->y, s2->w, buf); }
                        } else {
                            if (NSTI == 1 && wn < a.nitems) issue_interior(wn, 0);
                            if (wn + gridDim.x < a.nitems) { issue_small(wn + gridDim.x, buf); if (NSTI == 2) issue_interior(wn + gridDim.x, buf); }
                        }
                    }
                }
            };
            if constexpr (!MOO) release_buffers();
            if (scaled) {
#pragma unroll
                for (int c = 0; c < 12; c++) { acc[c].re = vmul(a.sigma, acc[c].re); acc[c].im = vmul(a.sigma, acc[c].im); }
            }
            if constexpr (MOO) {
                // out = M_oo^-1 res (closed form of DESIGN.md sec. 5.4), fused: the tile is transposed through the
                // interior buffer (rows = (site, component), padded by one group against bank conflicts), then one
                // thread per row walks s in registers and stores the row (contiguous in the output block).
                constexpr int VL = Prec<R>::VL;
                G* s_t = reinterpret_cast<G*>(smem + TG::HDR + ib * TG::INT_STRIDE);    // this item's interior buffer
                __syncthreads();                               // every warp is done reading the interior
#pragma unroll
                for (int c = 0; c < 12; c++) s_t[(ls * 12 + c) * (K + 1) + k] = pack(acc[c]);
                // When K divides 32 a site's rows are written and read back by threads of ONE warp: each warp solves the rows of its
                // own sites (32/K sites x 24 tasks) and the two hand-overs are warp barriers, not CTA barriers.
                constexpr bool WARP_LOCAL = (32 % K == 0);
                constexpr int TASKS = WARP_LOCAL ? (32 / K) * 24 : TS * 24;        // per warp | per CTA
                constexpr int TSTEP = WARP_LOCAL ? 32 : TG::THREADS;
                const int task0 = WARP_LOCAL ? (int)(threadIdx.x >> 5) * TASKS : 0;
                if constexpr (WARP_LOCAL) __syncwarp(); else __syncthreads();
                const R kappa = a.moo_kappa, v0scale = a.moo_v0scale, mass = a.mass;
                G* obase_t = a.out[pi] + (size_t)blk_index(gg * TS, r, a.nrhs, SH) * BS;   // the tile's blocks are one run
                // task = (row, real | imaginary part): TS*24 tasks = a whole number of passes of the CTA (3 for 32 sites x 256
                // threads) with Ls values in registers each; the two tasks of a row sit in neighbouring lanes, so a pair reads
                // and writes whole 16-byte groups
                using H = typename std::conditional<VL == 2, float2, double>::type;        // one part of a group
                const H* s_h = reinterpret_cast<const H*>(s_t);
                for (int tk = WARP_LOCAL ? (int)(threadIdx.x & 31) : (int)threadIdx.x; tk < TASKS; tk += TSTEP) {
                    const int task = task0 + tk;
                    const int row = task >> 1, part = task & 1;
                    const int c = row % 12;
                    const bool down = DAG ? (c >= 6) : (c < 6);
                    R b[LS];
#pragma unroll
                    for (int kk = 0; kk < K; kk++) {
                        const H g = s_h[(row * (K + 1) + (down ? kk : K - 1 - kk)) * 2 + part];
                        if constexpr (VL == 2) { b[2 * kk] = down ? g.x : g.y; b[2 * kk + 1] = down ? g.y : g.x; }
                        else b[kk] = g;
                    }
                    const R b0 = b[0];
                    b[0] = R(0);
#pragma unroll
                    for (int j = 1; j < LS; j++) b[j] = kappa * (b[j] + b[j - 1]);
                    const R v0 = v0scale * (b0 - mass * b[LS - 1]);
                    R pw = R(1);
#pragma unroll
                    for (int j = 0; j < LS; j++) { b[j] = fma(pw, v0, b[j]); pw *= kappa; }
                    // back into the same row of the transposition buffer (only this task touches its half of the row) ...
                    H* s_w = reinterpret_cast<H*>(s_t);
#pragma unroll
                    for (int kk = 0; kk < K; kk++) {
                        H g;
                        if constexpr (VL == 2) { g.x = down ? b[2 * kk] : b[2 * kk + 1]; g.y = down ? b[2 * kk + 1] : b[2 * kk]; }
                        else g = b[kk];
                        s_w[(row * (K + 1) + (down ? kk : K - 1 - kk)) * 2 + part] = g;
                    }
                }
                if constexpr (WARP_LOCAL) __syncwarp(); else __syncthreads();
                // ... and out in the lane layout: the same whole-line streaming stores as every other epilogue (storing the rows
                // straight from the tasks costs 16 half-used sectors per warp instruction: Schur K1 91 us instead of 7x us)
                {
                    G* o = obase_t + (size_t)ls * BS + k;
#pragma unroll
                    for (int c = 0; c < 12; c++) __stcs(o + c * K, s_t[(ls * 12 + c) * (K + 1) + k]);
                }
                release_buffers();                             // the reads of the buffer are complete (values consumed)
                continue;
            }
        }
        int ko = k;
        if constexpr (G5) {
            ko = K - 1 - k;
            // with the axpby epilogue its factor ax_a rides on the lane swap (two scalar multiplies into the swapped positions
            // instead of two register moves and a packed multiply)
#pragma unroll
            for (int c = 0; c < 12; c++) {
                if constexpr (AXPBY) {
                    const R sc = (c >= 6) ? -ax_a : ax_a;
                    acc[c].re = vswapmul(sc, acc[c].re); acc[c].im = vswapmul(sc, acc[c].im);
                } else {
                    const R sc = (c >= 6) ? R(-1) : R(1);          // exact; scalar multiplies into the swapped positions: MOV 173 -> 112
                    acc[c].re = vswapmul(sc, acc[c].re); acc[c].im = vswapmul(sc, acc[c].im);
                }
            }
            // res = (H_DW + shift) in: the input at the OUTPUT location is lane group K-1-k of this thread's own (site, rhs) block,
            // the lines the self term has just read (L1 hits).  The factored Chebyshev step of dwf_api.cu x_step uses it.
            if (SELF && a.g5_shift != R(0)) {
                const G* t = a.in_self[pi] + (size_t)blk * BS + ko;
                const R sh = AXPBY ? ax_a * a.g5_shift : a.g5_shift;
#pragma unroll
                for (int c = 0; c < 12; c++) {
                    const CV<V> tt = unpack(ldg_nc(t + c * K));
                    acc[c].re = vfma(sh, tt.re, acc[c].re); acc[c].im = vfma(sh, tt.im, acc[c].im);
                }
            }
        }
        const size_t obase = (size_t)blk * BS + ko;
        if constexpr (AXPBY) {
            const G* y = a.y[pi] + obase;
            const G* z = a.z[pi] + obase;
            if constexpr (!G5) {
#pragma unroll
                for (int c = 0; c < 12; c++) { acc[c].re = vmul(ax_a, acc[c].re); acc[c].im = vmul(ax_a, acc[c].im); }
            }
            if (a.ax_b != R(0)) {                              // a zero coefficient means "operand absent": it is not read
#pragma unroll
                for (int c = 0; c < 12; c++) {
                    const CV<V> yy = unpack(ldg_nc(y + c * K));
                    acc[c].re = vfma(a.ax_b, yy.re, acc[c].re); acc[c].im = vfma(a.ax_b, yy.im, acc[c].im);
                }
            }
            if (a.ax_c != R(0)) {
#pragma unroll
                for (int c = 0; c < 12; c++) {
                    const CV<V> zz = unpack(ld_plain(z + c * K));
                    acc[c].re = vfma(a.ax_c, zz.re, acc[c].re); acc[c].im = vfma(a.ax_c, zz.im, acc[c].im);
                }
            }
        }
        G* o = a.out[pi] + obase;
#pragma unroll
        for (int c = 0; c < 12; c++) __stcs(o + c * K, pack(acc[c]));          // streaming store: the output is not re-read by this launch
        if constexpr (NORM) {
            // |out|^2 of this warp's part of the item, fp64: fixed shuffle tree inside the warp, one partial per (item, warp)
            double sre = 0, sim = 0;
#pragma unroll
            for (int c = 0; c < 12; c++) acc_inner(sre, sim, acc[c], acc[c]);
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) sre += __shfl_xor_sync(0xffffffffu, sre, off);
            if ((threadIdx.x & 31) == 0) a.norm_partial[(size_t)(w - a.item0) * NWARPS + (threadIdx.x >> 5)] = sre;
        }
    }
    if (dyn) {                                                 // the last CTA to leave zeroes the item counter for the next launch
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            if (atomicAdd(a.dyn_counter + 1, 1u) == gridDim.x - 1) { a.dyn_counter[0] = 0u; a.dyn_counter[1] = 0u; __threadfence(); }
        }
    }
    if constexpr (NORM) {
        // the last CTA to arrive sums the (item, warp) partials in index order: deterministic, no extra launch
        __shared__ bool s_last;
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) s_last = (atomicAdd(a.ticket, 1u) == gridDim.x - 1);
        __syncthreads();
        if (s_last) {
            __threadfence();
            __shared__ double s_sum[TG::THREADS];
            // NWARPS is even and the slots are 16-byte aligned: 128-bit loads, 16 in flight per thread (the sum is one L2 round trip or
            // two at 16^3x32: 16k partials; fixed order per thread, then thread order)
            static_assert(NWARPS % 2 == 0, "pairs of partials");
            const long long n2 = (a.nitems - a.item0) * (NWARPS / 2);
            const double2* pp = reinterpret_cast<const double2*>(a.norm_partial);
            double t = 0;
#pragma unroll 16
            for (long long k = threadIdx.x; k < n2; k += TG::THREADS) { const double2 v = __ldcg(pp + k); t += v.x; t += v.y; }
            s_sum[threadIdx.x] = t;
            __syncthreads();
            if (threadIdx.x == 0) {
                double tot = 0;
                for (int k = 0; k < TG::THREADS; k++) tot += s_sum[k];
                *a.norm_out = tot;
                *a.ticket = 0u;
            }
        }
    }
}

}  // namespace dwf
