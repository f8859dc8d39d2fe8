// dwf_api.cu -- host side of libdwf: the C ABI of include/dwf.h, index tables, kernel dispatch and
// the two drivers (Chebyshev recurrence, red-black CGNR) that only enqueue kernels.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <algorithm>
#include <array>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <numeric>
#include <vector>

#include "../../include/dwf.h"
#include "dwf_aux.cuh"
#include "dwf_hop.cuh"
#include "dwf_tile.cuh"

using namespace dwf;

static const int MAX_RED_BLOCKS = 2048;
static const int MAX_NRHS = 64;
static const int SCAL_DOUBLES = 1 << 16;

struct dwf_ctx {
    int L[4], Ls, prec;
    double M5, mass;
    long long V4, V4h;
    cudaStream_t stream;
    cudaStream_t cap_stream;   // private stream used only to capture the CG loop into a CUDA graph
    void* gauge;          // native links [2][V4h][4][18] reals
    void* glinks;         // gathered, (-1/2)-scaled links for the tiled stencil (tile_sites != 0)
    int* nbr;             // [2][V4h][8]
    int* lex;             // [2][V4h]
    int* inv_lex;         // [V4]: lexicographic site -> index within its parity (built on first use by dwf_convert)
    bool have_gauge;
    void* ws; size_t ws_bytes;
    double* partial;      // reduction partials [blocks][nrhs][2]
    size_t partial_doubles;   // its size: covers blas_blocks(nrhs) * nrhs * 2 for every nrhs <= MAX_NRHS
    unsigned* ticket;     // CTA completion counter of the fused norm (zero between launches)
    double* scal;         // device scalars (reduction results, CG history)
    double* scal_host;    // pinned mirror
    int sm_count, device;
    size_t l2_bytes;      // cudaDevAttrL2CacheSize (picks the t-extent of the lattice blocks, build_tables)
    bool cheb_factored;   // DWF_CHEB_FACTORED: dwf_chebyshev steps as alpha (H - c)(H + c) t instead of the literal alpha H(H t) - beta t
    bool no_dyn;          // DWF_NO_DYN: static instead of dynamic item assignment in the tiled stencil
    bool no_fuse_moo, no_fuse_norm;   // DWF_NO_FUSE_MOOINV / DWF_NO_FUSE_NORM, read once at dwf_create (the unfused reference path)
    int cg_graph;         // DWF_CG_GRAPH, read once at dwf_create: 0 never, 1 always, unset (-1): launch-bound sizes only
    // the instantiated CUDA graph of the last CG solve and the arguments it was captured for (re-launched when they recur)
    long long cg_launches;
    cudaGraphExec_t cg_exec; const void* cg_b; void* cg_x; void* cg_ws; size_t cg_ws_bytes; int cg_iters, cg_nrhs, cg_kind;
    long long blk_sites;  // sites per parity in one lattice block of the native site order
    int blk_t;            // t-extent of a lattice block; 0 when the block order is not lexicographic with t slowest (no t-layers)
    cudaStream_t io_in, io_out;          // dwf_apply_host pipeline: H2D and D2H streams, created on first use
    cudaEvent_t io_ev[2 * 16 + 1];       //   chunk c arrived / chunk c exported / the handle's stream reached the call
    int tile_sites;       // sites per parity in one tile of the native site order (0: lattice is not made of whole tiles)
    int sg_shift;         // block order [site group][rhs][site in group]: log2(group size)
    bool rhs_batch;       // one rhs-major stencil launch for a batch of right-hand sides (off: DWF_RHS_LOOP=1 or static item assignment)
    int rhs_chunk;        // right-hand sides per stencil launch
    long long launches;
    char err[256];
};


#define FAIL(h, code, ...) do { snprintf((h)->err, sizeof((h)->err), __VA_ARGS__); return (code); } while (0)
#define CUDA_TRY(h, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) \
    FAIL(h, DWF_ECUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); } while (0)
#define LAUNCH_CHECK(h) do { (h)->launches++; cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) \
    FAIL(h, DWF_ECUDA, "kernel launch failed: %s", cudaGetErrorString(e_)); } while (0)

static inline size_t real_bytes(const dwf_ctx* h) { return h->prec == DWF_F32 ? 4 : 8; }
static inline int vl(const dwf_ctx* h) { return h->prec == DWF_F32 ? 2 : 1; }
static inline size_t half_bytes(const dwf_ctx* h, int nrhs) {
    return (size_t)h->V4h * 24 * (size_t)h->Ls * (size_t)nrhs * real_bytes(h);
}
static inline long long half_groups(const dwf_ctx* h, int nrhs) {
    return h->V4h * 12 * ((long long)nrhs * h->Ls / vl(h));
}
static inline int block_groups(const dwf_ctx* h) { return 12 * h->Ls / vl(h); }   // groups per (site, rhs) block
static inline int run_groups(const dwf_ctx* h) { return block_groups(h) << h->sg_shift; }   // groups per contiguous run of one rhs

// BLAS-1 launch geometry: (blocks * 256) % period == 0 (period = groups per site group = run_groups * nrhs) so that each
// thread keeps one rhs for its whole grid-stride loop.  `unit` may exceed MAX_RED_BLOCKS (wide blocks x many rhs):
// h->partial is sized for that at dwf_create.
static long long blas_unit(long long period) { return period / std::gcd(period, 256LL); }
static long long blas_blocks_for(long long unit, long long want) {
    long long blocks = std::max<long long>(unit, (want / unit) * unit);
    if (blocks > MAX_RED_BLOCKS) blocks = std::max<long long>(unit, (MAX_RED_BLOCKS / unit) * unit);
    return blocks;
}

// ------------------------------------------------------------------------------------------------
// Index tables.  Native site order within a parity: 4D blocks of BLK^4 sites in lexicographic block
// order, lexicographic inside a block (locality for L1/L2: DESIGN.md sec. 4.1); tables make the order
// a free choice.  DWF_BLOCK="bx,by,bz,bt" overrides the default.
// ------------------------------------------------------------------------------------------------
static void build_tables(dwf_ctx* h, std::vector<int>& lex, std::vector<int>& nbr) {
    const int* L = h->L;
    int B[4] = {4, 4, 4, 4};      // outer block: unit of the parity interleave, L2 locality
    int T[4] = {4, 4, 2, 2};      // inner tile : 32 sites per parity = what one CTA of the tiled stencil works on
    // the tile interior of one rhs must fit shared memory twice per SM: 16-site tiles for wide blocks
    // (measured at 48^3x96 fp32 Ls 24: 32-site tiles x 1 CTA/SM 20.2 ms per apply, 16-site tiles x 2 CTAs/SM 24.2 ms)
    if ((size_t)h->Ls * 24 * real_bytes(h) > 2304) T[1] = 2;
    // small lattices: fewer 32-site tiles than two per SM leave most of the GPU idle in every launch -- 16-site tiles double the
    // work items (measured on B200, 8^4 x 16 fp32 red-black CG: 23.6k -> 28.5k iterations/s)
    if (h->V4h / 32 < 2LL * h->sm_count) T[1] = 2;
    // Blocks are swept x fastest, t slowest, so the -t halo of a block layer is re-read one layer later.  When two layers of
    // t-extent 2 (input + output + gathered links) fit L2 the thin layer keeps that halo resident: measured on B200 at 16^3x32x16,
    // block 4,4,4,2 against 4,4,4,4: D_DW fp32 130.5 -> 127.0 us, fp64 304 -> 281 us, H_DW fp64 nrhs 12 3.81 -> 3.67 ms.  When a layer is
    // far larger than L2 (48^3x96x24: 510 MB) every t face misses anyway and the taller block halves the faces: 4,4,4,4 21.4 ms,
    // 4,4,4,2 25.1 ms, 4,4,4,8 23.7 ms (larger blocks lengthen the y/z reuse distance instead).
    bool big_layers;
    {
        const double layer2 = (double)L[0] * L[1] * L[2] * 2 * ((double)h->Ls * 24 * 2 + 2 * 72) * real_bytes(h);
        big_layers = 2 * layer2 > (double)h->l2_bytes;
        if (!big_layers) B[3] = 2;
    }
    auto parse = [](const char* name, int* v) {
        if (const char* env = getenv(name)) { int b[4]; if (sscanf(env, "%d,%d,%d,%d", &b[0], &b[1], &b[2], &b[3]) == 4) for (int i = 0; i < 4; i++) v[i] = b[i]; }
    };
    parse("DWF_BLOCK", B); parse("DWF_TILE", T);
    for (int i = 0; i < 4; i++) if (B[i] < 1 || L[i] % B[i] != 0) B[i] = L[i];   // fall back to no blocking
    if ((B[0] * B[1] * B[2] * B[3]) % 2 != 0) B[0] = L[0];                      // blocks must hold both parities equally
    for (int i = 0; i < 4; i++) if (T[i] < 1 || B[i] % T[i] != 0) T[i] = B[i];
    if ((T[0] * T[1] * T[2] * T[3]) % 2 != 0) for (int i = 0; i < 4; i++) T[i] = B[i];
    const long long V4 = h->V4, V4h = h->V4h;
    h->blk_sites = (long long)B[0] * B[1] * B[2] * B[3] / 2;
    { const char* o = getenv("DWF_BLOCK_ORDER"); const bool lexo = o ? !strcmp(o, "lex") : !big_layers; h->blk_t = (lexo && L[3] % B[3] == 0) ? B[3] : 0; }   // lexicographic block order: t-layers of blocks are contiguous site ranges
    const int tsites = T[0] * T[1] * T[2] * T[3] / 2;
    bool whole = true;
    for (int i = 0; i < 4; i++) whole = whole && (L[i] % T[i] == 0);
    h->tile_sites = (whole && (tsites == 16 || tsites == 32 || tsites == 64)) ? tsites : 0;
    h->sg_shift = h->tile_sites == 64 ? 6 : h->tile_sites == 32 ? 5 : h->tile_sites == 16 ? 4 : 0;
    if (getenv("DWF_NO_TILE")) h->tile_sites = 0;             // keeps the block order, uses the generic kernel
    lex.assign(2 * V4h, 0);
    std::vector<int> idx_of(V4);                                                // lex site -> index within its parity
    long long cnt[2] = {0, 0};
    int nb[4], nt[4]; for (int i = 0; i < 4; i++) { nb[i] = L[i] / B[i]; nt[i] = B[i] / T[i]; }
    // Order of the lattice blocks: lexicographic (x fastest).  It re-reads the +-t halo of a block one 3-D slab of blocks later;
    // when that slab no longer fits L2 the z and t halos come from DRAM twice (48^3 x 96 x 24: DRAM reads 2.15x the algorithmic
    // bytes, ncu).  Two alternatives are kept behind DWF_BLOCK_ORDER for measurement and are NOT the default: "panel" (the (x,y,z)
    // cross-section cut into panels of px x py x pz blocks whose slab fits DWF_L2_BUDGET_MB, t swept inside each panel) and "morton"
    // (Z-order curve).  Measured on B200: panel 23.5 ms against 21.0 ms per D_DW apply at 48^3 x 96 x 24 (the kernel is bound by its
    // LSU wavefronts there, 68 %, not by DRAM), +-1 % at 16^3 x 32 in either precision; morton +-2 %.
    std::vector<std::array<int, 4>> blocks;
    for (int bt = 0; bt < nb[3]; bt++) for (int bz = 0; bz < nb[2]; bz++) for (int by = 0; by < nb[1]; by++) for (int bx = 0; bx < nb[0]; bx++)
        blocks.push_back({bx, by, bz, bt});
    {
        const char* ord = getenv("DWF_BLOCK_ORDER");
        // Lattices whose t-layers are far larger than L2 (48^3x96x24: 510 MB): panels (the (x,y,z) cross-section cut so that a panel's
        // layer fits half the L2, t swept inside each panel) keep the z and t halos resident.  Measured on B200 with the dynamic item
        // assignment of the tiled kernel: D_DW 19.1 ms lexicographic, 18.3-18.7 ms panels of 16-128 MB, 18.4 ms Morton.  (With the
        // static assignment every order but the lexicographic one DOUBLED the DRAM reads: the CTAs drift apart and the window of items
        // in flight outgrows the L2.)  "lex" forces the lexicographic order.
        if (!ord && big_layers) ord = "panel";
        const double block_mb = (double)B[0] * B[1] * B[2] * B[3] * ((double)h->Ls * 24 * 2 + 72) * real_bytes(h) / 1e6;   // in + out + links
        double budget_mb = (double)h->l2_bytes / 2e6;           // half the L2 (DWF_L2_BUDGET_MB overrides: tuning)
        if (const char* e = getenv("DWF_L2_BUDGET_MB")) budget_mb = std::max(1.0, atof(e));
        if (ord && !strcmp(ord, "morton")) {
            auto code = [](const std::array<int, 4>& b) {
                unsigned long long c = 0;
                for (int bit = 0; bit < 16; bit++) for (int d = 0; d < 4; d++) c |= (unsigned long long)((b[d] >> bit) & 1) << (4 * bit + d);
                return c;
            };
            std::stable_sort(blocks.begin(), blocks.end(), [&](const std::array<int, 4>& x, const std::array<int, 4>& y) { return code(x) < code(y); });
        } else if (ord && !strcmp(ord, "panel")) {
            // panel extents: start from the whole cross-section and halve the largest extent (keeping divisibility) until it fits
            int P[3] = {nb[0], nb[1], nb[2]};
            while ((double)P[0] * P[1] * P[2] * block_mb > budget_mb) {
                int best = -1;
                for (int d = 0; d < 3; d++) if (P[d] > 1 && (best < 0 || P[d] > P[best])) best = d;
                if (best < 0) break;
                int q = P[best] - 1;                            // largest smaller divisor of nb[best]
                while (q > 1 && nb[best] % q != 0) q--;
                P[best] = q;
            }
            auto key = [&](const std::array<int, 4>& b) {
                const long long panel = (b[0] / P[0]) + (long long)(nb[0] / P[0]) * ((b[1] / P[1]) + (long long)(nb[1] / P[1]) * (b[2] / P[2]));
                const long long inside = (b[0] % P[0]) + (long long)P[0] * ((b[1] % P[1]) + (long long)P[1] * (b[2] % P[2]));
                return (panel * nb[3] + b[3]) * ((long long)P[0] * P[1] * P[2]) + inside;
            };
            std::stable_sort(blocks.begin(), blocks.end(), [&](const std::array<int, 4>& x, const std::array<int, 4>& y) { return key(x) < key(y); });
        }
    }
    for (const auto& bb : blocks) { const int bx = bb[0], by = bb[1], bz = bb[2], bt = bb[3];
      for (int tt = 0; tt < nt[3]; tt++) for (int tz = 0; tz < nt[2]; tz++) for (int ty = 0; ty < nt[1]; ty++) for (int tx = 0; tx < nt[0]; tx++) {
        const int o[4] = {bx * B[0] + tx * T[0], by * B[1] + ty * T[1], bz * B[2] + tz * T[2], bt * B[3] + tt * T[3]};
        for (int t = o[3]; t < o[3] + T[3]; t++) for (int z = o[2]; z < o[2] + T[2]; z++)
            for (int y = o[1]; y < o[1] + T[1]; y++) for (int x = o[0]; x < o[0] + T[0]; x++) {
                const int p = (x + y + z + t) & 1;
                const long long lx = x + (long long)L[0] * (y + (long long)L[1] * (z + (long long)L[2] * t));
                lex[p * V4h + cnt[p]] = (int)lx;
                idx_of[lx] = (int)cnt[p];
                cnt[p]++;
            }
      }
    }
    nbr.assign(2 * V4h * 8, 0);
    for (int p = 0; p < 2; p++) for (long long i = 0; i < V4h; i++) {
        long long lx = lex[p * V4h + i];
        int c[4]; long long r = lx;
        for (int d = 0; d < 4; d++) { c[d] = (int)(r % L[d]); r /= L[d]; }
        for (int mu = 0; mu < 4; mu++) for (int dir = 0; dir < 2; dir++) {
            int n[4] = {c[0], c[1], c[2], c[3]};
            n[mu] = (c[mu] + (dir == 0 ? 1 : L[mu] - 1)) % L[mu];
            const long long nl = n[0] + (long long)L[0] * (n[1] + (long long)L[1] * (n[2] + (long long)L[2] * n[3]));
            nbr[(p * V4h + i) * 8 + 2 * mu + dir] = idx_of[nl];
        }
    }
}

extern "C" int dwf_create(const int L[4], int Ls, double M5, double mass, int precision, dwf_handle* out) {
    if (!out) return DWF_EINVAL;
    *out = nullptr;
    if (!L) return DWF_EINVAL;
    for (int i = 0; i < 4; i++) if (L[i] < 4 || (L[i] & 1)) return DWF_EINVAL;
    if (Ls < 2 || Ls > 64 || (Ls & 1)) return DWF_EINVAL;
    if (precision != DWF_F32 && precision != DWF_F64) return DWF_EINVAL;
    if (M5 == 5.0 || !std::isfinite(M5) || !std::isfinite(mass)) return DWF_EINVAL;
    if (1.0 + mass * std::pow(5.0 - M5, -(double)Ls) == 0.0) return DWF_EINVAL;
    const long long V4 = (long long)L[0] * L[1] * L[2] * L[3];
    if (V4 / 2 * 8 >= (1LL << 31)) return DWF_EUNSUPPORTED;
    dwf_ctx* h = new (std::nothrow) dwf_ctx();
    if (!h) return DWF_ENOMEM;
    memset(h, 0, sizeof(*h));
    for (int i = 0; i < 4; i++) h->L[i] = L[i];
    h->Ls = Ls; h->prec = precision; h->M5 = M5; h->mass = mass;
    h->V4 = V4; h->V4h = V4 / 2;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        delete h; return DWF_ECUDA;
    }
    h->device = dev;
    { int l2 = 0; if (cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev) != cudaSuccess || l2 <= 0) l2 = 64 << 20; h->l2_bytes = (size_t)l2; }
    h->no_fuse_moo = getenv("DWF_NO_FUSE_MOOINV") != nullptr;
    h->no_fuse_norm = getenv("DWF_NO_FUSE_NORM") != nullptr;
    h->no_dyn = getenv("DWF_NO_DYN") != nullptr;
    h->cheb_factored = getenv("DWF_CHEB_FACTORED") != nullptr;
    { const char* genv = getenv("DWF_CG_GRAPH"); h->cg_graph = genv ? atoi(genv) : -1; }
    std::vector<int> lex, nbr;
    build_tables(h, lex, nbr);
    h->rhs_chunk = 1;      // measured on B200 (16^3x32x16 fp32): 1 is fastest (132 us per rhs at nrhs 12; 4: 142 us): a chunk of c rhs needs c slabs of the lattice in L2
    if (const char* env = getenv("DWF_RHS_CHUNK")) h->rhs_chunk = std::max(1, atoi(env));
    h->rhs_batch = getenv("DWF_RHS_LOOP") == nullptr && !h->no_dyn;
    h->partial_doubles = std::max((size_t)MAX_RED_BLOCKS * MAX_NRHS * 2, (size_t)(h->V4h * (Ls / vl(h)) / 32 + 64));   // BLAS-1 partials | fused-norm partials
    for (int n = 1; n <= MAX_NRHS; n++) {                    // worst case of blas_blocks(): one unit of blocks larger than MAX_RED_BLOCKS
        const long long unit = blas_unit((long long)run_groups(h) * n);
        h->partial_doubles = std::max(h->partial_doubles, (size_t)blas_blocks_for(unit, MAX_RED_BLOCKS) * n * 2);
    }
    const size_t gbytes = (size_t)2 * h->V4h * 72 * real_bytes(h);
    const size_t glbytes = (size_t)2 * h->V4h * (144 * real_bytes(h) + 16);
    bool ok = cudaMalloc(&h->gauge, gbytes) == cudaSuccess
           && (h->tile_sites == 0 || (cudaMalloc(&h->glinks, glbytes) == cudaSuccess && cudaMemset(h->glinks, 0, glbytes) == cudaSuccess))
           && cudaMalloc((void**)&h->nbr, nbr.size() * sizeof(int)) == cudaSuccess
           && cudaMalloc((void**)&h->lex, lex.size() * sizeof(int)) == cudaSuccess
           && cudaMalloc((void**)&h->partial, h->partial_doubles * sizeof(double)) == cudaSuccess
           && cudaMalloc((void**)&h->scal, SCAL_DOUBLES * sizeof(double)) == cudaSuccess
           && cudaMalloc((void**)&h->ticket, 64) == cudaSuccess && cudaMemset(h->ticket, 0, 64) == cudaSuccess
           && cudaMallocHost((void**)&h->scal_host, SCAL_DOUBLES * sizeof(double)) == cudaSuccess
           && cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaMemcpy(h->nbr, nbr.data(), nbr.size() * sizeof(int), cudaMemcpyHostToDevice) == cudaSuccess
            && cudaMemcpy(h->lex, lex.data(), lex.size() * sizeof(int), cudaMemcpyHostToDevice) == cudaSuccess;
    if (!ok) { cudaGetLastError(); dwf_destroy(h); return DWF_ENOMEM; }
    *out = h;
    return DWF_OK;
}

extern "C" int dwf_destroy(dwf_handle h) {
    if (!h) return DWF_EINVAL;
    cudaFree(h->gauge); cudaFree(h->glinks); cudaFree(h->inv_lex); cudaFree(h->nbr); cudaFree(h->lex); cudaFree(h->partial); cudaFree(h->scal); cudaFree(h->ticket);
    if (h->scal_host) cudaFreeHost(h->scal_host);
    if (h->cg_exec) cudaGraphExecDestroy(h->cg_exec);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    if (h->io_in) { cudaStreamDestroy(h->io_in); cudaStreamDestroy(h->io_out); for (cudaEvent_t e : h->io_ev) if (e) cudaEventDestroy(e); }
    delete h;
    return DWF_OK;
}

extern "C" int dwf_set_stream(dwf_handle h, void* s) { if (!h) return DWF_EINVAL; h->stream = (cudaStream_t)s; return DWF_OK; }
extern "C" const char* dwf_last_error(dwf_handle h) { return h ? h->err : "null handle"; }
extern "C" long long dwf_launch_count(dwf_handle h) { return h ? h->launches : -1; }

extern "C" size_t dwf_field_bytes(dwf_handle h, int nrhs, int half) {
    if (!h || nrhs < 1) return 0;
    return half ? half_bytes(h, nrhs) : 2 * half_bytes(h, nrhs);
}
extern "C" size_t dwf_workspace_bytes(dwf_handle h, int nrhs) {
    if (!h || nrhs < 1) return 0;
    return 12 * half_bytes(h, nrhs) + 256;         // dwf_solve_mixed: 8 (dwf_solve) + 2 full fields
}
extern "C" int dwf_set_workspace(dwf_handle h, void* p, size_t n) {
    if (!h) return DWF_EINVAL;
    if (p && ((uintptr_t)p & 15)) FAIL(h, DWF_EINVAL, "workspace must be 16-byte aligned");
    h->ws = p; h->ws_bytes = p ? n : 0;
    return DWF_OK;
}
static int need_ws(dwf_ctx* h, size_t bytes) {
    if (!h->ws || h->ws_bytes < bytes)
        FAIL(h, DWF_ENOWORKSPACE, "workspace of %zu bytes needed, %zu set (dwf_set_workspace)", bytes, h->ws_bytes);
    return DWF_OK;
}
static int check_field(dwf_ctx* h, const void* p, const char* name) {
    if (!p) FAIL(h, DWF_EINVAL, "%s is NULL", name);
    if ((uintptr_t)p & 15) FAIL(h, DWF_EINVAL, "%s is not 16-byte aligned", name);
    return DWF_OK;
}

// ------------------------------------------------------------------------------------------------
extern "C" int dwf_set_gauge(dwf_handle h, const void* U) {
    if (!h) return DWF_EINVAL;
    if (int rc = check_field(h, U, "U_canonical_dev")) return rc;
    const long long n = 2 * h->V4h * 36;
    const long long spatial = (long long)h->L[0] * h->L[1] * h->L[2];
    const unsigned blocks = (unsigned)((n + 255) / 256);
    if (h->prec == DWF_F32) reorder_gauge_kernel<float><<<blocks, 256, 0, h->stream>>>((const float*)U, (float*)h->gauge, h->lex, h->V4h, h->V4, spatial, h->L[3]);
    else                    reorder_gauge_kernel<double><<<blocks, 256, 0, h->stream>>>((const double*)U, (double*)h->gauge, h->lex, h->V4h, h->V4, spatial, h->L[3]);
    LAUNCH_CHECK(h);
    if (h->glinks) {
        const long long m = 2 * h->V4h * 144;
        const unsigned gb = (unsigned)((m + 255) / 256);
        if (h->prec == DWF_F32) gather_links_kernel<float><<<gb, 256, 0, h->stream>>>((const float*)h->gauge, (float*)h->glinks, h->nbr, h->V4h, TileLinks<float>::SITE);
        else                    gather_links_kernel<double><<<gb, 256, 0, h->stream>>>((const double*)h->gauge, (double*)h->glinks, h->nbr, h->V4h, TileLinks<double>::SITE);
        LAUNCH_CHECK(h);
    }
    h->have_gauge = true;
    return DWF_OK;
}

// site0 .. site1: the sites (native order, per parity) this launch converts; site1 = 0: all
template <typename R, bool IMPORT>
static int reorder_spinor(dwf_ctx* h, const void* canon_in, void* canon_out, void* native, int nrhs, int parity,
                          long long site0 = 0, long long site1 = 0) {
    using G = typename Prec<R>::G;
    const long long per_parity = half_groups(h, nrhs);
    G* n0; G* n1; const int* l0; const int* l1; unsigned ny;
    if (parity < 0) { n0 = (G*)native; n1 = (G*)native + per_parity; l0 = h->lex; l1 = h->lex + h->V4h; ny = 2; }
    else            { n0 = n1 = (G*)native; l0 = l1 = h->lex + (size_t)parity * h->V4h; ny = 1; }
    if (site1 == 0) site1 = h->V4h;
    const long long pairs = (site1 - site0) * nrhs;                              // one warp per (site, rhs) block
    dim3 grid((unsigned)((pairs + 3) / 4), ny);
    const size_t dsm = 4 * 24 * (size_t)h->Ls * sizeof(R);
    reorder_spinor_kernel<R, IMPORT><<<grid, 128, dsm, h->stream>>>((const R*)canon_in, (R*)canon_out, n0, n1, l0, l1, h->V4h, h->V4, h->Ls, nrhs, h->sg_shift,
                                                                    site0 * nrhs, site1 * nrhs);
    LAUNCH_CHECK(h);
    return DWF_OK;
}

extern "C" int dwf_import(dwf_handle h, const void* canonical, void* native, int nrhs, int parity) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS || parity < -1 || parity > 1) FAIL(h, DWF_EINVAL, "bad nrhs/parity");
    if (int rc = check_field(h, canonical, "canonical")) return rc;
    if (int rc = check_field(h, native, "native")) return rc;
    return h->prec == DWF_F32 ? reorder_spinor<float, true>(h, canonical, nullptr, native, nrhs, parity)
                              : reorder_spinor<double, true>(h, canonical, nullptr, native, nrhs, parity);
}
extern "C" int dwf_export(dwf_handle h, const void* native, void* canonical, int nrhs, int parity) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS || parity < -1 || parity > 1) FAIL(h, DWF_EINVAL, "bad nrhs/parity");
    if (int rc = check_field(h, canonical, "canonical")) return rc;
    if (int rc = check_field(h, native, "native")) return rc;
    return h->prec == DWF_F32 ? reorder_spinor<float, false>(h, nullptr, canonical, (void*)native, nrhs, parity)
                              : reorder_spinor<double, false>(h, nullptr, canonical, (void*)native, nrhs, parity);
}

// ------------------------------------------------------------------------------------------------
// Stencil dispatch
// ------------------------------------------------------------------------------------------------
enum HopMode { HM_HOP, HM_HOP_SELF, HM_HOP_SELF_G5, HM_HOP_SELF_G5_AXPBY, HM_SELF, HM_HOP_MOOINV /* tiled only */,
               HM_HOP_SELF_AXPBY_NORM /* tiled only: CG residual update fused into the adjoint Schur K2 */ };

struct HopCall {            // precision-independent description of one launch
    int mode; bool dag;
    int nslots, parity0;    // output parities: parity0 (, parity0^1)
    const void* in_hop[2]; const void* in_self[2]; void* out[2]; const void* y[2]; const void* z[2];
    double c_hop, mass, ax_a, ax_b, ax_c;
    int nrhs;
    double* norm_out;       // tiled HM_HOP_SELF (not dag) and HM_HOP_SELF_AXPBY_NORM, nrhs = 1: also *norm_out = |out|^2 (device), summed
                            // inside the launch (dwf_tile.cuh NORM epilogue)
    const double* ax_num; const double* ax_den;   // HM_HOP_SELF_AXPBY_NORM: ax_a = -(*ax_num / *ax_den), read on the device
    long long site0, site1;  // output sites (native order, per parity) of this launch, whole lattice blocks; site1 = 0: all
    double g5_shift;         // HM_HOP_SELF_G5*: out = (H_DW + g5_shift) in [then the axpby epilogue]
};

// Is the tiled persistent stencil (dwf_tile.cuh) instantiated for this handle?  Lattice made of whole tiles, Ls 16 (16- or
// 32-site tiles) or Ls 24 (16-site tiles; 32-site tiles in fp32), item index within 32 bits.
static bool tiled_ok(const dwf_ctx* h) {
    if (!h->glinks || !h->tile_sites) return false;
    if (h->tile_sites == 64 && !(h->Ls == 16 && h->prec == DWF_F32)) return false;
    if (!(h->Ls == 16 || (h->Ls == 24 && (h->tile_sites == 16 || h->prec == DWF_F32)))) return false;
    return 2 * (h->V4h / h->tile_sites + h->blk_sites) * (long long)h->rhs_chunk < (1LL << 31);
}

// Partial launches (HopCall::site0/site1) cover whole parity-interleave chunks: this many sites per parity
static long long partial_unit(const dwf_ctx* h) {
    const int K = h->Ls / vl(h);
    const long long GS = tiled_ok(h) ? h->tile_sites : std::min(HOP_THREADS / 8, HOP_THREADS / K);
    return std::max<long long>(1, h->blk_sites / GS) * GS;
}

template <typename R>
static int launch_hop_t(dwf_ctx* h, const HopCall& k) {
    using G = typename Prec<R>::G;
    HopArgs<R> a;
    for (int s = 0; s < 2; s++) {
        const int p = (k.parity0 + s) & 1;
        a.in_hop[s] = (const G*)k.in_hop[s]; a.in_self[s] = (const G*)k.in_self[s]; a.out[s] = (G*)k.out[s];
        a.y[s] = (const G*)k.y[s]; a.z[s] = (const G*)k.z[s];
        a.nbr[s] = h->nbr + (size_t)p * h->V4h * 8;
        a.gauge[s] = (const R*)h->gauge + (size_t)s * h->V4h * 72;      // gauge[] is indexed by PARITY
    }
    a.V4h = h->V4h; a.Ls = h->Ls; a.nrhs = k.nrhs;
    a.parity0 = k.parity0; a.nslots = k.nslots;
    a.c_hop = (R)k.c_hop; a.c_diag = (R)(5.0 - h->M5); a.mass = (R)k.mass;
    a.ax_a = (R)k.ax_a; a.ax_b = (R)k.ax_b; a.ax_c = (R)k.ax_c; a.g5_shift = (R)k.g5_shift;
    const int K = h->Ls / Prec<R>::VL;
    // tiled persistent stencil (dwf_tile.cuh): lattice made of whole tiles, compile-time Ls, a hop to do
    const int TS = (k.mode != HM_SELF && tiled_ok(h) && h->V4h * (long long)k.nrhs < (1LL << 31)) ? h->tile_sites : 0;   // 32-bit block indices in the tiled kernel
    a.sg_shift = h->sg_shift;
    a.GS = TS ? TS : std::min(HOP_THREADS / 8, HOP_THREADS / K);                                   // sites per CTA
    a.ngroups = (h->V4h + a.GS - 1) / a.GS;
    a.chunk_groups = std::max<long long>(1, h->blk_sites / a.GS);             // parity interleave unit = one lattice block
    long long groups = a.ngroups;
    if (k.nslots == 2) groups = 2 * ((a.ngroups + a.chunk_groups - 1) / a.chunk_groups) * a.chunk_groups;
    long long group0 = 0;                                                       // first site group (CTA of the generic kernel / tile) of a partial launch
    if (k.site1) {
        const long long unit = a.chunk_groups * a.GS;                           // sites per parity-interleave chunk
        if (k.site0 % unit || k.site1 % unit || k.site1 > h->V4h) FAIL(h, DWF_EINVAL, "partial launch: site range must be whole lattice blocks");
        group0 = k.site0 / a.GS * k.nslots; groups = k.site1 / a.GS * k.nslots;
    }
    cudaStream_t st = h->stream;
    const size_t lsite = 144 * sizeof(R) + 16;
    a.glinks[0] = (const R*)h->glinks;
    a.glinks[1] = (const R*)((const char*)h->glinks + (size_t)h->V4h * lsite);
    a.sigma = (R)(-2.0 * k.c_hop);                                             // links carry the factor -1/2
    a.norm_partial = h->partial; a.norm_out = k.norm_out; a.ticket = h->ticket;
    a.dyn_counter = h->no_dyn ? nullptr : h->ticket + 2;
    a.ax_num = k.ax_num; a.ax_den = k.ax_den;
    {
        const double kappa = 1.0 / (5.0 - h->M5);
        a.moo_kappa = (R)kappa; a.moo_v0scale = (R)(kappa / (1.0 + k.mass * std::pow(kappa, (double)h->Ls)));
    }
    if (k.mode == HM_HOP_MOOINV && !TS) FAIL(h, DWF_EINVAL, "fused hop + M_oo^-1 needs the tiled kernel");
#define HOPK(LS, DAG, HOP, SELF, G5, AX) hop_kernel<R, LS, DAG, HOP, SELF, G5, AX><<<grid, HOP_THREADS, 0, st>>>(a)
#define TILEK(LS, TSV, DAG, SELF, G5, AX, MOO, NRM) do { \
        using TG = TileGeom<R, LS, TSV>; \
        auto kern = hop_tile_kernel<R, LS, TSV, DAG, true, SELF, G5, AX, MOO, NRM>; \
        static unsigned long long attr_done = 0;              /* per kernel instantiation: devices whose attribute is set */ \
        if (!((attr_done >> (h->device & 63)) & 1ull)) { \
            cudaError_t e_ = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TG::SMEM_BYTES); \
            if (e_ != cudaSuccess) FAIL(h, DWF_ECUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e_)); \
            attr_done |= 1ull << (h->device & 63); \
        } \
        const long long ctas = std::min<long long>(a.nitems - a.item0, (long long)h->sm_count * TG::MIN_CTAS); \
        if (a.nitems - a.item0 <= 2 * ctas) a.dyn_counter = nullptr;   /* launch-bound sizes: nothing to hand out, skip the counter traffic */ \
        kern<<<(unsigned)ctas, TG::THREADS, TG::SMEM_BYTES, st>>>(a); } while (0)
#define HOPM(LS) \
    switch (k.mode) { \
        case HM_HOP:               if (k.dag) HOPK(LS, true, true, false, false, false); else HOPK(LS, false, true, false, false, false); break; \
        case HM_HOP_SELF:          if (k.dag) HOPK(LS, true, true, true, false, false);  else HOPK(LS, false, true, true, false, false); break; \
        case HM_HOP_SELF_G5:       HOPK(LS, false, true, true, true, false); break; \
        case HM_HOP_SELF_G5_AXPBY: HOPK(LS, false, true, true, true, true); break; \
        case HM_SELF:              if (k.dag) HOPK(LS, true, false, true, false, false); else HOPK(LS, false, false, true, false, false); break; \
        default: FAIL(h, DWF_EINVAL, "bad hop mode"); \
    }
#define TILEM(LS, TSV) \
    switch (k.mode) { \
        case HM_HOP:               if (k.dag) TILEK(LS, TSV, true, false, false, false, false, false); else TILEK(LS, TSV, false, false, false, false, false, false); break; \
        case HM_HOP_MOOINV:        if (k.dag) TILEK(LS, TSV, true, false, false, false, true, false); else TILEK(LS, TSV, false, false, false, false, true, false); break; \
        case HM_HOP_SELF:          if (k.dag) TILEK(LS, TSV, true, true, false, false, false, false); \
                                   else if (k.norm_out) TILEK(LS, TSV, false, true, false, false, false, true); \
                                   else TILEK(LS, TSV, false, true, false, false, false, false); break; \
        case HM_HOP_SELF_G5:       TILEK(LS, TSV, false, true, true, false, false, false); break; \
        case HM_HOP_SELF_G5_AXPBY: TILEK(LS, TSV, false, true, true, true, false, false); break; \
        case HM_HOP_SELF_AXPBY_NORM: TILEK(LS, TSV, true, true, false, true, false, true); break; \
        default: FAIL(h, DWF_EINVAL, "bad hop mode"); \
    }
    if ((k.norm_out || k.mode == HM_HOP_SELF_AXPBY_NORM) && (!TS || k.nrhs != 1)) FAIL(h, DWF_EINVAL, "fused norm needs the tiled kernel and nrhs = 1");
    // Right-hand sides are processed in chunks (one launch each) so that the working set of a chunk keeps
    // the L2 reuse of the single-rhs case; CTAs of one chunk run tile-major, rhs-minor.
    // Default (rhs_chunk 1): ONE launch for the whole batch with the items ordered rhs-major -- every rhs sweeps the lattice on its own
    // (DESIGN.md sec. 5.3), without the ramp-up, the partly filled last round and the launch gap of one launch per rhs.  It needs the
    // dynamic item assignment of the tiled kernel: with the static one the CTAs drift apart over the 330 rounds of a 24-rhs launch
    // and it is 15 % SLOWER than one launch per rhs.  DWF_RHS_LOOP=1: one launch per rhs; DWF_RHS_CHUNK=c > 1: tile-major chunks of c rhs.
    const bool batch = TS && h->rhs_chunk == 1 && h->rhs_batch && k.nrhs > 1 && !k.site1 && !k.norm_out && groups * k.nrhs < (1LL << 31);
    const int RC = batch ? k.nrhs : h->rhs_chunk;
    a.items_per_rhs = batch ? (unsigned)groups : 0u;
    for (int r0 = 0; r0 < k.nrhs; r0 += RC) {
        a.r0 = r0; a.rn = std::min(RC, k.nrhs - r0);
        a.item0 = group0 * a.rn; a.nitems = groups * a.rn;
        dim3 grid((unsigned)((groups - group0) * a.rn));
        // compile-time Ls for the production sizes (tiled when the lattice allows), runtime Ls otherwise
        if (h->Ls == 16)      { if (TS == 64) { if constexpr (sizeof(R) == 4) { TILEM(16, 64) } } else if (TS == 32) { TILEM(16, 32) } else if (TS == 16) { TILEM(16, 16) } else { HOPM(16) } }
        else if (h->Ls == 24) { if (TS == 16) { TILEM(24, 16) } else if (TS == 32) { if constexpr (sizeof(R) == 4) { TILEM(24, 32) } } else { HOPM(24) } }
        else { HOPM(0) }
        LAUNCH_CHECK(h);
    }
#undef TILEM
#undef TILEK
#undef HOPM
#undef HOPK
    return DWF_OK;
}
static int launch_hop(dwf_ctx* h, const HopCall& k) {
    return h->prec == DWF_F32 ? launch_hop_t<float>(h, k) : launch_hop_t<double>(h, k);
}

template <typename R, bool DAG>
static int launch_mooinv_t(dwf_ctx* h, const void* in, void* out, int nrhs, double mass) {
    using G = typename Prec<R>::G;
    const double kappa = 1.0 / (5.0 - h->M5);
    const double v0scale = kappa / (1.0 + mass * std::pow(kappa, (double)h->Ls));
    const long long threads = h->V4h * 12 * nrhs;
    const unsigned blocks = (unsigned)((threads + 127) / 128);
#define MOOK(LS) mooinv_kernel<R, LS, DAG><<<blocks, 128, 0, h->stream>>>((const G*)in, (G*)out, h->V4h, nrhs, h->sg_shift, (R)kappa, (R)mass, (R)v0scale)
    switch (h->Ls) {
        case 4: MOOK(4); break;   case 8: MOOK(8); break;   case 12: MOOK(12); break;
        case 16: MOOK(16); break; case 24: MOOK(24); break; case 32: MOOK(32); break;
        default: FAIL(h, DWF_EUNSUPPORTED, "M_oo^-1 is instantiated for Ls in {4,8,12,16,24,32}, got %d", h->Ls);
    }
#undef MOOK
    LAUNCH_CHECK(h);
    return DWF_OK;
}
static int launch_mooinv(dwf_ctx* h, const void* in, void* out, int nrhs, double mass, bool dag) {
    if (h->prec == DWF_F32) return dag ? launch_mooinv_t<float, true>(h, in, out, nrhs, mass) : launch_mooinv_t<float, false>(h, in, out, nrhs, mass);
    return dag ? launch_mooinv_t<double, true>(h, in, out, nrhs, mass) : launch_mooinv_t<double, false>(h, in, out, nrhs, mass);
}

// full-lattice operator:  out_p = c_hop hop(in_{1-p}) [+ self(in_p)] for both parities, one launch
static int full_op(dwf_ctx* h, int mode, bool dag, double c_hop, double mass, const void* in, void* out, int nrhs,
                   double ax_a = 0, const void* y = nullptr, double ax_b = 0, const void* z = nullptr, double ax_c = 0,
                   long long site0 = 0, long long site1 = 0, double g5_shift = 0.0) {
    const size_t hb = half_bytes(h, nrhs);
    HopCall k{};
    k.mode = mode; k.dag = dag; k.nslots = 2; k.parity0 = 0; k.nrhs = nrhs;
    for (int p = 0; p < 2; p++) {
        k.in_hop[p] = (const char*)in + (size_t)(1 - p) * hb;
        k.in_self[p] = (const char*)in + (size_t)p * hb;
        k.out[p] = (char*)out + (size_t)p * hb;
        k.y[p] = y ? (const char*)y + (size_t)p * hb : nullptr;
        k.z[p] = z ? (const char*)z + (size_t)p * hb : nullptr;
    }
    k.c_hop = c_hop; k.mass = mass; k.ax_a = ax_a; k.ax_b = ax_b; k.ax_c = ax_c;
    k.site0 = site0; k.site1 = site1; k.g5_shift = g5_shift;
    return launch_hop(h, k);
}

// Schur operator on even half fields:  tmp_o = M_oo^-1 Dhop_oe in ;
// out = M_ee in - 1/4 Dhop_eo tmp_o     [M_eo = M_oe = -1/2 Dhop].  dag: every factor adjoint.
// norm_out != NULL (nrhs = 1, not dag): also *norm_out = |out|^2 on the device; fused into K2 when the tiled kernel applies.
static int reduce_to(dwf_ctx* h, bool norm, const void* x, const void* y, int nrhs, int half, double* dev_out, int ostride, int ncomp);
// Can the |out|^2 of a stencil launch be summed inside the launch (tiled kernel, one rhs, partials fit the scratch)?
static bool norm_fusable(const dwf_ctx* h, int nrhs) {
    return tiled_ok(h) && !h->no_fuse_moo && !h->no_fuse_norm && nrhs == 1
        && (size_t)(h->V4h * (h->Ls / vl(h)) / 32) <= h->partial_doubles;       // one partial per (tile, warp) of a half-lattice launch
}
struct SchurFuse {          // dag only (CG, q = M^dag w): r <- r - (num/den) q instead of storing q, and *norm_out = |r|^2
    void* r; const double* num; const double* den;
};
static int schur_op(dwf_ctx* h, bool dag, const void* in, void* out, void* tmp, int nrhs, double* norm_out = nullptr,
                    const SchurFuse* fuse = nullptr) {
    // K1: tmp_o = M_oo^-1 Dhop_oe in -- one launch when the tiled kernel applies (M_oo^-1 fused as its epilogue)
    const bool fused = tiled_ok(h) && !h->no_fuse_moo;
    HopCall k1{};
    k1.mode = fused ? HM_HOP_MOOINV : HM_HOP; k1.dag = dag; k1.nslots = 1; k1.parity0 = 1; k1.nrhs = nrhs;
    k1.in_hop[0] = in; k1.out[0] = tmp; k1.c_hop = 1.0; k1.mass = h->mass;
    if (int rc = launch_hop(h, k1)) return rc;
    if (!fused) { if (int rc = launch_mooinv(h, tmp, tmp, nrhs, h->mass, dag)) return rc; }
    HopCall k2{};
    k2.mode = HM_HOP_SELF; k2.dag = dag; k2.nslots = 1; k2.parity0 = 0; k2.nrhs = nrhs;
    k2.in_hop[0] = tmp; k2.in_self[0] = in; k2.out[0] = out; k2.c_hop = -0.25; k2.mass = h->mass;
    if (fuse) {                                               // out = r - alpha (M_pc^dag in), |out|^2: one launch, q never stored
        if (!dag || !norm_out || !norm_fusable(h, nrhs)) FAIL(h, DWF_EINVAL, "fused residual update: adjoint Schur, tiled kernel, nrhs = 1");
        k2.mode = HM_HOP_SELF_AXPBY_NORM; k2.out[0] = fuse->r; k2.z[0] = fuse->r; k2.y[0] = fuse->r;
        k2.ax_a = 0.0; k2.ax_b = 0.0; k2.ax_c = 1.0; k2.ax_num = fuse->num; k2.ax_den = fuse->den; k2.norm_out = norm_out;
        return launch_hop(h, k2);
    }
    const bool fuse_norm = norm_out && !dag && norm_fusable(h, nrhs);
    if (fuse_norm) k2.norm_out = norm_out;
    if (int rc = launch_hop(h, k2)) return rc;
    if (!norm_out || fuse_norm) return DWF_OK;
    return reduce_to(h, true, out, nullptr, nrhs, 1, norm_out, 1, 1);
}

static int apply_checked(dwf_ctx* h, int op, const void* in, void* out, int nrhs) {
    const bool dag = (op & DWF_DAGGER) != 0;
    const int base = op & ~DWF_DAGGER;
    switch (base) {
        case DWF_DHOP: return full_op(h, HM_HOP, dag, 1.0, h->mass, in, out, nrhs);
        case DWF_DDW:  return full_op(h, HM_HOP_SELF, dag, -0.5, h->mass, in, out, nrhs);
        case DWF_DPV:  return full_op(h, HM_HOP_SELF, dag, -0.5, 1.0, in, out, nrhs);
        case DWF_HDW:  return full_op(h, HM_HOP_SELF_G5, false, -0.5, h->mass, in, out, nrhs);
        case DWF_SCHUR_EO: {
            if (int rc = need_ws(h, half_bytes(h, nrhs))) return rc;
            return schur_op(h, dag, in, out, h->ws, nrhs);
        }
        case DWF_MEE: {
            HopCall k{};
            k.mode = HM_SELF; k.dag = dag; k.nslots = 1; k.parity0 = 0; k.nrhs = nrhs;
            k.in_self[0] = in; k.out[0] = out; k.mass = h->mass;
            return launch_hop(h, k);
        }
        case DWF_MOOINV: return launch_mooinv(h, in, out, nrhs, h->mass, dag);
        case DWF_SCHUR_EO_ALT: {                              // 1 - M_ee^-1 M_eo M_oo^-1 M_oe = 1 - 1/4 M_ee^-1 Dhop_eo M_oo^-1 Dhop_oe
            // adjoint: 1 - 1/4 Dhop_oe^dag (M_oo^dag)^-1 Dhop_eo^dag (M_ee^dag)^-1  (the factors in reverse order)
            const size_t hb = half_bytes(h, nrhs);
            if (int rc = need_ws(h, 2 * hb)) return rc;
            void* t1 = h->ws; void* t2 = (char*)h->ws + hb;
            const bool fusedk = tiled_ok(h) && !h->no_fuse_moo;
            auto hop_moo = [&](int parity_out, const void* src, void* dst, bool with_moo) -> int {   // dst_p = [M_pp^-1] Dhop src_{1-p}
                HopCall k{}; k.mode = (with_moo && fusedk) ? HM_HOP_MOOINV : HM_HOP; k.dag = dag; k.nslots = 1; k.parity0 = parity_out; k.nrhs = nrhs;
                k.in_hop[0] = src; k.out[0] = dst; k.c_hop = 1.0; k.mass = h->mass;
                if (int rc = launch_hop(h, k)) return rc;
                if (with_moo && !fusedk) return launch_mooinv(h, dst, dst, nrhs, h->mass, dag);
                return DWF_OK;
            };
            if (!dag) {
                if (int rc = hop_moo(1, in, t1, true)) return rc;                  // t1_o = M_oo^-1 Dhop_oe in
                if (int rc = hop_moo(0, t1, t2, true)) return rc;                  // t2_e = M_ee^-1 Dhop_eo t1
            } else {
                if (int rc = launch_mooinv(h, in, t2, nrhs, h->mass, true)) return rc;   // t2_e = (M_ee^dag)^-1 in
                if (int rc = hop_moo(1, t2, t1, true)) return rc;                  // t1_o = (M_oo^dag)^-1 Dhop_eo^dag t2   [Dhop_eo^dag maps even -> odd]
                if (int rc = hop_moo(0, t1, t2, false)) return rc;                 // t2_e = Dhop_oe^dag t1
            }
            CUDA_TRY(h, cudaMemcpyAsync(out, in, hb, cudaMemcpyDeviceToDevice, h->stream));
            double coef[2 * MAX_NRHS];
            for (int q = 0; q < nrhs; q++) { coef[2 * q] = -0.25; coef[2 * q + 1] = 0.0; }
            return dwf_axpy(h, coef, t2, out, nrhs, 1);
        }
        case DWF_MPVDAG_M: {                                  // D_PV^dag D_DW (dag: D_DW^dag D_PV): two stencil launches through the workspace
            if (int rc = need_ws(h, 2 * half_bytes(h, nrhs))) return rc;
            if (int rc = full_op(h, HM_HOP_SELF, false, -0.5, dag ? 1.0 : h->mass, in, h->ws, nrhs)) return rc;
            return full_op(h, HM_HOP_SELF, true, -0.5, dag ? h->mass : 1.0, h->ws, out, nrhs);
        }
        default: FAIL(h, DWF_EINVAL, "unknown op %d", op);
    }
}

extern "C" int dwf_apply(dwf_handle h, int op, const void* in, void* out, int nrhs) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS) FAIL(h, DWF_EINVAL, "nrhs must be in [1,%d]", MAX_NRHS);
    if (int rc = check_field(h, in, "in")) return rc;
    if (int rc = check_field(h, out, "out")) return rc;
    if (in == out) FAIL(h, DWF_EINVAL, "in == out: the stencil is not in-place safe");
    const int base = op & ~DWF_DAGGER;
    if (base != DWF_MEE && base != DWF_MOOINV && !h->have_gauge) FAIL(h, DWF_ENOGAUGE, "dwf_set_gauge has not been called");
    return apply_checked(h, op, in, out, nrhs);
}

// ------------------------------------------------------------------------------------------------
// Chebyshev driver:  X = alpha H^2 - beta, alpha = 2/(hi-lo), beta = (hi+lo)/(hi-lo)
//   t_1 = alpha H(H t_0) - beta t_0 ;  t_{k+1} = 2 alpha H(H t_k) - 2 beta t_k - t_{k-1}
// Each step = two stencil launches; the second carries the three-term recurrence in its epilogue and
// overwrites t_{k-1} in place.  Odd t_k live in buffer A, even ones in B; A/B are chosen so that
// t_order lands in `out`.
// ------------------------------------------------------------------------------------------------
// One step of a recurrence in X = alpha H^2 - beta (H = H_DW), two stencil launches through the scratch field w:
//     dst = coef (alpha H^2 - beta) tk + cz z            (z may alias dst; cz = 0: no z)
// Literal form (default; SURVEY 8(a) a8, 6 field passes):   w = H tk ;  dst = coef alpha H w - coef beta tk + cz z.
// Factored form (DWF_CHEB_FACTORED=1, 5 field passes):  alpha H^2 - beta = alpha (H - c)(H + c),  c = sqrt(beta / alpha)  [H is hermitian
// and commutes with c]:   w = (H + c) tk ;  dst = coef alpha (H - c) w + cz z.   The shift rides in the G5 epilogue (the input at the output
// location = another lane group of the block the self term has just read), so the second launch no longer reads tk.  Measured on B200:
// order-64 Chebyshev on 24 vectors 485 -> 474 ms; error against the oracle 9.0e-6 instead of 3.3e-6 (fp32), 1.3e-14 instead of 2.7e-14 (fp64).
// Opt-in: the bench line and its roofline keep the literal form that SURVEY's algorithmic byte count (144R per 5D site and order) describes.
static int x_step(dwf_ctx* h, const void* tk, void* w, void* dst, int nrhs, double coef, double alpha, double beta, const void* z, double cz) {
    if (h->cheb_factored && beta > 0.0 && alpha > 0.0) {
        const double c = std::sqrt(beta / alpha);
        if (int rc = full_op(h, HM_HOP_SELF_G5, false, -0.5, h->mass, tk, w, nrhs, 0, nullptr, 0, nullptr, 0, 0, 0, +c)) return rc;
        return full_op(h, HM_HOP_SELF_G5_AXPBY, false, -0.5, h->mass, w, dst, nrhs, coef * alpha, z ? z : tk, 0.0, z ? z : tk, z ? cz : 0.0, 0, 0, -c);
    }
    if (int rc = full_op(h, HM_HOP_SELF_G5, false, -0.5, h->mass, tk, w, nrhs)) return rc;
    return full_op(h, HM_HOP_SELF_G5_AXPBY, false, -0.5, h->mass, w, dst, nrhs, coef * alpha, tk, -coef * beta, z ? z : tk, z ? cz : 0.0);
}

extern "C" int dwf_chebyshev(dwf_handle h, int order, double lo, double hi, const void* in, void* out, int nrhs) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS) FAIL(h, DWF_EINVAL, "nrhs must be in [1,%d]", MAX_NRHS);
    if (order < 0 || !(hi > lo)) FAIL(h, DWF_EINVAL, "need order >= 0 and hi > lo");
    if (int rc = check_field(h, in, "in")) return rc;
    if (int rc = check_field(h, out, "out")) return rc;
    if (in == out) FAIL(h, DWF_EINVAL, "in == out");
    if (!h->have_gauge) FAIL(h, DWF_ENOGAUGE, "dwf_set_gauge has not been called");
    const size_t fb = 2 * half_bytes(h, nrhs);
    if (order == 0) { CUDA_TRY(h, cudaMemcpyAsync(out, in, fb, cudaMemcpyDeviceToDevice, h->stream)); return DWF_OK; }
    if (int rc = need_ws(h, 2 * fb)) return rc;
    void* w = h->ws;
    void* other = (char*)h->ws + fb;
    void* A = (order & 1) ? out : other;      // holds t_1, t_3, ...
    void* B = (order & 1) ? other : out;      // holds t_2, t_4, ...
    const double alpha = 2.0 / (hi - lo), beta = (hi + lo) / (hi - lo);
    // t_1 = alpha H H t_0 - beta t_0
    if (int rc = x_step(h, in, w, A, nrhs, 1.0, alpha, beta, nullptr, 0.0)) return rc;
    const void* tkm1 = in; void* tk = A;
    for (int k = 1; k < order; k++) {
        void* dst = (k == 1) ? B : (void*)tkm1;           // t_{k+1} overwrites t_{k-1} (except t_0 = user input)
        if (int rc = x_step(h, tk, w, dst, nrhs, 2.0, alpha, beta, tkm1, -1.0)) return rc;
        tkm1 = tk; tk = dst;
    }
    return DWF_OK;
}

// ------------------------------------------------------------------------------------------------
// Subspace generation by Chebyshev filtering (eq. 34-37).
//   first pass : v = T_m(2(H^2 - lambda_lo)/(lambda_max - lambda_lo) - 1) eta                 (eq. 34, reading R10)
//   then ONE recurrence in X' = 2 H^2/lambda_max - 1 started from v, emitting
//   phi_k = T_{k Delta}(X') v  for k = 0 .. nvec-1  ("all for the cost of the highest order", L229; eq. 37)
// phi: nvec consecutive full native fields of nrhs right-hand sides each.  Workspace: 3 full fields.
// ------------------------------------------------------------------------------------------------
extern "C" int dwf_chebyshev_subspace(dwf_handle h, int m, double lambda_lo, double lambda_max, int delta, int nvec,
                                      const void* eta, void* phi, int nrhs) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS) FAIL(h, DWF_EINVAL, "nrhs must be in [1,%d]", MAX_NRHS);
    if (m < 0 || delta < 1 || nvec < 1 || !(lambda_max > lambda_lo) || !(lambda_lo >= 0.0)) FAIL(h, DWF_EINVAL, "need m >= 0, delta >= 1, nvec >= 1, 0 <= lambda_lo < lambda_max");
    if (int rc = check_field(h, eta, "eta")) return rc;
    if (int rc = check_field(h, phi, "phi")) return rc;
    if (eta == phi) FAIL(h, DWF_EINVAL, "eta == phi");
    if (!h->have_gauge) FAIL(h, DWF_ENOGAUGE, "dwf_set_gauge has not been called");
    const size_t fb = 2 * half_bytes(h, nrhs);
    if (int rc = need_ws(h, 3 * fb)) return rc;
    // first pass straight into phi_0 (dwf_chebyshev uses workspace fields 0 and 1)
    if (int rc = dwf_chebyshev(h, m, lambda_lo, lambda_max, eta, phi, nrhs)) return rc;
    // Outside [lambda_lo, lambda_max] T_m grows as cosh(m acosh|x|) (Fig. 2: 1e8 for the paper's parameters, but
    // 1e137 for m = 600, lambda_lo = 4): no normalisation is applied (R14), so an overflow of the field's precision is
    // reported instead of returning inf/nan vectors.
    auto check_finite = [&](const void* f, const char* what) -> int {
        double n2[MAX_NRHS];
        if (int rc = dwf_norm2(h, f, n2, nrhs, 0)) return rc;
        for (int q = 0; q < nrhs; q++) if (!std::isfinite(n2[q]))
            FAIL(h, DWF_ERANGE, "%s overflowed %s (rhs %d): lower m or raise lambda_lo, or use an fp64 handle", what, h->prec == DWF_F32 ? "fp32" : "fp64", q);
        return DWF_OK;
    };
    if (int rc = check_finite(phi, "first-pass filter T_m")) return rc;
    if (nvec == 1) return DWF_OK;
    void* w = h->ws; void* A = (char*)h->ws + fb; void* B = (char*)h->ws + 2 * fb;
    const double alpha = 2.0 / lambda_max, beta = 1.0;                          // X' = alpha H^2 - beta
    const void* t0 = phi;
    if (int rc = full_op(h, HM_HOP_SELF_G5, false, -0.5, h->mass, t0, w, nrhs)) return rc;
    if (int rc = full_op(h, HM_HOP_SELF_G5_AXPBY, false, -0.5, h->mass, w, A, nrhs, alpha, t0, -beta, t0, 0.0)) return rc;
    const void* tkm1 = t0; void* tk = A;
    const int last = (nvec - 1) * delta;
    for (int k = 1; ; k++) {                                                   // tk = t_k
        if (k % delta == 0)
            CUDA_TRY(h, cudaMemcpyAsync((char*)phi + (size_t)(k / delta) * fb, tk, fb, cudaMemcpyDeviceToDevice, h->stream));
        if (k == last) break;
        void* dst = (k == 1) ? B : (void*)tkm1;                                 // t_{k+1} overwrites t_{k-1} (t_0 = phi_0 is kept)
        if (int rc = full_op(h, HM_HOP_SELF_G5, false, -0.5, h->mass, tk, w, nrhs)) return rc;
        if (int rc = full_op(h, HM_HOP_SELF_G5_AXPBY, false, -0.5, h->mass, w, dst, nrhs, 2.0 * alpha, tk, -2.0 * beta, tkm1, -1.0)) return rc;
        tkm1 = tk; tk = dst;
    }
    return check_finite((char*)phi + (size_t)(nvec - 1) * fb, "second-pass recurrence");   // lambda_max below the true one: |x| > 1
}

// Chebyshev smoother (eq. 24-25):
//   out = [ c_0/2 + sum_{j=1..N} c_j T_j(2(M^dag M - a)/(b - a) - 1) ] M^dag r ,   M = D_DW,  M^dag M = H_DW^2,
//   c_j = (2/N) sum_{k<N} f(y(cos theta_k)) cos(j theta_k),  f(y) = 1/y,  theta_k = pi (k + 1/2)/N,
//   y(x) = ((b - a) x + (b + a))/2.
// v = M^dag r by the adjoint stencil, then the three-term recurrence of dwf_chebyshev with a forward summation
// (one axpy per order).  Workspace: 4 full fields (v, w, t_odd, t_even).
extern "C" int dwf_chebyshev_smoother(dwf_handle h, int N, double a, double b, const void* r, void* out, int nrhs) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS) FAIL(h, DWF_EINVAL, "nrhs must be in [1,%d]", MAX_NRHS);
    if (N < 1 || N > 4096 || !(b > a) || !(a > 0.0)) FAIL(h, DWF_EINVAL, "need 1 <= N <= 4096 and 0 < a < b");
    if (int rc = check_field(h, r, "r")) return rc;
    if (int rc = check_field(h, out, "out")) return rc;
    if (r == out) FAIL(h, DWF_EINVAL, "r == out");
    if (!h->have_gauge) FAIL(h, DWF_ENOGAUGE, "dwf_set_gauge has not been called");
    const size_t fb = 2 * half_bytes(h, nrhs);
    if (int rc = need_ws(h, 4 * fb)) return rc;
    std::vector<double> c(N + 1);
    const double pi = 3.14159265358979323846;
    for (int j = 0; j <= N; j++) {
        double acc = 0;
        for (int k = 0; k < N; k++) {
            const double th = pi * (k + 0.5) / N;
            const double y = 0.5 * ((b - a) * std::cos(th) + (b + a));
            acc += std::cos(j * th) / y;
        }
        c[j] = 2.0 * acc / N;
    }
    void* v = h->ws; void* w = (char*)h->ws + fb; void* A = (char*)h->ws + 2 * fb; void* B = (char*)h->ws + 3 * fb;
    double coef[2 * MAX_NRHS];
    auto add = [&](double cj, const void* t) -> int {                          // out += cj t
        for (int q = 0; q < nrhs; q++) { coef[2 * q] = cj; coef[2 * q + 1] = 0.0; }
        return dwf_axpy(h, coef, t, out, nrhs, 0);
    };
    if (int rc = full_op(h, HM_HOP_SELF, true, -0.5, h->mass, r, v, nrhs)) return rc;           // v = D_DW^dag r
    CUDA_TRY(h, cudaMemsetAsync(out, 0, fb, h->stream));
    if (int rc = add(0.5 * c[0], v)) return rc;
    // c_N = (2/N) sum_k cos(N theta_k)/y_k vanishes identically (cos(N theta_k) = cos(pi (k + 1/2)) = 0): the sum of eq. 24
    // stops at j = N-1 and the last recurrence step (two operator applies) is not needed.
    if (N == 1) return DWF_OK;
    const double alpha = 2.0 / (b - a), beta = (b + a) / (b - a);
    if (int rc = full_op(h, HM_HOP_SELF_G5, false, -0.5, h->mass, v, w, nrhs)) return rc;
    if (int rc = full_op(h, HM_HOP_SELF_G5_AXPBY, false, -0.5, h->mass, w, A, nrhs, alpha, v, -beta, v, 0.0)) return rc;
    if (int rc = add(c[1], A)) return rc;
    const void* tkm1 = v; void* tk = A;
    for (int k = 1; k < N - 1; k++) {
        void* dst = (k == 1) ? B : (void*)tkm1;
        if (int rc = full_op(h, HM_HOP_SELF_G5, false, -0.5, h->mass, tk, w, nrhs)) return rc;
        if (int rc = full_op(h, HM_HOP_SELF_G5_AXPBY, false, -0.5, h->mass, w, dst, nrhs, 2.0 * alpha, tk, -2.0 * beta, tkm1, -1.0)) return rc;
        tkm1 = tk; tk = dst;
        if (int rc = add(c[k + 1], tk)) return rc;
    }
    return DWF_OK;
}

// lambda_max(H_DW^2) by the power method (L225), nrhs = 1.  v holds the start vector on entry and the last
// iterate on return.  Iteration i: u = H v; lambda_i = |u|^2/|v|^2 (Rayleigh quotient of H^2); v <- H u / lambda_i
// (keeps |v| = O(1)).  lambda_hist_host (may be NULL) receives the `iters` quotients; returns the last in *lambda_host.
// Workspace: 2 full fields.
extern "C" int dwf_power_lambda_max(dwf_handle h, int iters, void* v, double* lambda_host, double* lambda_hist_host) {
    if (!h) return DWF_EINVAL;
    if (iters < 1 || !lambda_host) FAIL(h, DWF_EINVAL, "need iters >= 1 and lambda_host");
    if (int rc = check_field(h, v, "v")) return rc;
    if (!h->have_gauge) FAIL(h, DWF_ENOGAUGE, "dwf_set_gauge has not been called");
    const size_t fb = 2 * half_bytes(h, 1);
    if (int rc = need_ws(h, 2 * fb)) return rc;
    void* u = h->ws; void* vn = (char*)h->ws + fb;
    void* cur = v; void* nxt = vn;
    double lam = 0.0;
    for (int i = 0; i < iters; i++) {
        if (int rc = full_op(h, HM_HOP_SELF_G5, false, -0.5, h->mass, cur, u, 1)) return rc;
        double nu = 0, nv = 0;
        if (int rc = reduce_to(h, true, u, nullptr, 1, 0, h->scal, 1, 1)) return rc;
        if (int rc = reduce_to(h, true, cur, nullptr, 1, 0, h->scal + 1, 1, 1)) return rc;
        CUDA_TRY(h, cudaMemcpyAsync(h->scal_host, h->scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(h, cudaStreamSynchronize(h->stream));
        nu = h->scal_host[0]; nv = h->scal_host[1];
        if (!(nv > 0.0) || !(nu > 0.0)) FAIL(h, DWF_EINVAL, "power method: zero vector");
        lam = nu / nv;
        if (lambda_hist_host) lambda_hist_host[i] = lam;
        if (int rc = full_op(h, HM_HOP_SELF_G5_AXPBY, false, -0.5, h->mass, u, nxt, 1, 1.0 / lam, u, 0.0, u, 0.0)) return rc;
        std::swap(cur, nxt);
    }
    if (cur != v) CUDA_TRY(h, cudaMemcpyAsync(v, cur, fb, cudaMemcpyDeviceToDevice, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    *lambda_host = lam;
    return DWF_OK;
}

// ------------------------------------------------------------------------------------------------
// BLAS-1
// ------------------------------------------------------------------------------------------------
static unsigned blas_blocks(const dwf_ctx* h, long long ngroups, long long period) {
    const long long want = std::min<long long>((ngroups + 255) / 256, (long long)h->sm_count * 8);
    return (unsigned)blas_blocks_for(blas_unit(period), want);
}

static int reduce_to(dwf_ctx* h, bool norm, const void* x, const void* y, int nrhs, int half, double* dev_out, int ostride, int ncomp) {
    const long long ng = half_groups(h, nrhs) * (half ? 1 : 2);
    const int BS = run_groups(h);
    const unsigned blocks = blas_blocks(h, ng, (long long)BS * nrhs);
    if (h->prec == DWF_F32) {
        if (norm) inner_kernel<float, true><<<blocks, 256, 0, h->stream>>>((const float4*)x, nullptr, ng, BS, nrhs, h->partial);
        else      inner_kernel<float, false><<<blocks, 256, 0, h->stream>>>((const float4*)x, (const float4*)y, ng, BS, nrhs, h->partial);
    } else {
        if (norm) inner_kernel<double, true><<<blocks, 256, 0, h->stream>>>((const double2*)x, nullptr, ng, BS, nrhs, h->partial);
        else      inner_kernel<double, false><<<blocks, 256, 0, h->stream>>>((const double2*)x, (const double2*)y, ng, BS, nrhs, h->partial);
    }
    LAUNCH_CHECK(h);
    reduce_final_kernel<<<nrhs, 256, 0, h->stream>>>(h->partial, (int)blocks, nrhs, dev_out, ostride, ncomp);
    LAUNCH_CHECK(h);
    return DWF_OK;
}

extern "C" int dwf_axpy(dwf_handle h, const double* a_host, const void* x, void* y, int nrhs, int half) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS || !a_host) FAIL(h, DWF_EINVAL, "bad nrhs or a_host");
    if (int rc = check_field(h, x, "x")) return rc;
    if (int rc = check_field(h, y, "y")) return rc;
    RhsCoef a;
    for (int r = 0; r < nrhs; r++) { a.re[r] = a_host[2 * r]; a.im[r] = a_host[2 * r + 1]; }
    const long long ng = half_groups(h, nrhs) * (half ? 1 : 2);
    const int BS = run_groups(h);
    const unsigned blocks = blas_blocks(h, ng, (long long)BS * nrhs);
    if (h->prec == DWF_F32) axpy_kernel<float><<<blocks, 256, 0, h->stream>>>((const float4*)x, (float4*)y, ng, BS, nrhs, a);
    else                    axpy_kernel<double><<<blocks, 256, 0, h->stream>>>((const double2*)x, (double2*)y, ng, BS, nrhs, a);
    LAUNCH_CHECK(h);
    return DWF_OK;
}

extern "C" int dwf_inner(dwf_handle h, const void* x, const void* y, double* out_host, int nrhs, int half) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS || !out_host) FAIL(h, DWF_EINVAL, "bad nrhs or out_host");
    if (int rc = check_field(h, x, "x")) return rc;
    if (int rc = check_field(h, y, "y")) return rc;
    if (int rc = reduce_to(h, false, x, y, nrhs, half, h->scal, 2, 2)) return rc;
    CUDA_TRY(h, cudaMemcpyAsync(h->scal_host, h->scal, 2 * nrhs * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    memcpy(out_host, h->scal_host, 2 * nrhs * sizeof(double));
    return DWF_OK;
}

extern "C" int dwf_norm2(dwf_handle h, const void* x, double* out_host, int nrhs, int half) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS || !out_host) FAIL(h, DWF_EINVAL, "bad nrhs or out_host");
    if (int rc = check_field(h, x, "x")) return rc;
    if (int rc = reduce_to(h, true, x, nullptr, nrhs, half, h->scal, 1, 1)) return rc;
    CUDA_TRY(h, cudaMemcpyAsync(h->scal_host, h->scal, nrhs * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    memcpy(out_host, h->scal_host, nrhs * sizeof(double));
    return DWF_OK;
}

// ------------------------------------------------------------------------------------------------
// dwf_norm2_static: |x|^2 per right-hand side with NO allocation anywhere on its path (callers under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc).  Same two kernels and launch geometry as dwf_norm2; the per-block partials go
// to a file-scope __device__ array instead of the handle's cudaMalloc'ed scratch, the result to a DEVICE pointer (no host
// synchronisation).  The array is DWF_STATIC_SCRATCH_DOUBLES doubles = 256 KB, held by every GPU that loads the library until the
// process exits.  Every call on a device shares it: the partial slots a call reads are all written by that call first (nothing
// has to start at zero), but two calls that overlap on the GPU (different streams / handles) race on it.
// ------------------------------------------------------------------------------------------------
#define DWF_STATIC_SCRATCH_DOUBLES 32768
static __device__ __align__(256) double g_norm2_scratch[DWF_STATIC_SCRATCH_DOUBLES];
// In host code the name above is a host-side stand-in, not a device address: the address is asked for once per device.
static double* g_norm2_scratch_ptr[64];

extern "C" int dwf_norm2_static(dwf_handle h, const void* x, double* out_dev, int nrhs, int half) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS || !out_dev) FAIL(h, DWF_EINVAL, "bad nrhs or out_dev");
    if (int rc = check_field(h, x, "x")) return rc;
    int dev = -1;
    CUDA_TRY(h, cudaGetDevice(&dev));
    if (dev != h->device || dev < 0 || dev >= 64) FAIL(h, DWF_EINVAL, "the handle's device (%d) must be the current device (%d)", h->device, dev);
    if (!g_norm2_scratch_ptr[dev]) {                         // set-up, once per device, with that device current
        double* ptr = nullptr;
        CUDA_TRY(h, cudaGetSymbolAddress((void**)&ptr, g_norm2_scratch));
        if (!ptr) FAIL(h, DWF_ECUDA, "cudaGetSymbolAddress returned a null address");
        g_norm2_scratch_ptr[dev] = ptr;
    }
    double* partial = g_norm2_scratch_ptr[dev];
    const long long ng = half_groups(h, nrhs) * (half ? 1 : 2);
    const int BS = run_groups(h);
    const unsigned blocks = blas_blocks(h, ng, (long long)BS * nrhs);
    const size_t need = (size_t)blocks * nrhs * 2;
    if (need > (size_t)DWF_STATIC_SCRATCH_DOUBLES)
        FAIL(h, DWF_EUNSUPPORTED, "dwf_norm2_static: %zu doubles of scratch needed (%u blocks x %d rhs x 2), the static maximum is %d: use fewer right-hand sides per call or dwf_norm2",
             need, blocks, nrhs, DWF_STATIC_SCRATCH_DOUBLES);
    if (h->prec == DWF_F32) inner_kernel<float, true><<<blocks, 256, 0, h->stream>>>((const float4*)x, nullptr, ng, BS, nrhs, partial);
    else                    inner_kernel<double, true><<<blocks, 256, 0, h->stream>>>((const double2*)x, nullptr, ng, BS, nrhs, partial);
    LAUNCH_CHECK(h);
    reduce_final_kernel<<<nrhs, 256, 0, h->stream>>>(partial, (int)blocks, nrhs, out_dev, 1, 1);
    LAUNCH_CHECK(h);
    return DWF_OK;
}

// ------------------------------------------------------------------------------------------------
// Red-black CGNR driver.  Host loop that only enqueues; alpha and beta are
// computed on the device from reduction results kept in h->scal: hist[k] = |r_k|^2 at scal[k],
// <p_k, A p_k> = |M p_k|^2 at scal[iters+1+k].
// ------------------------------------------------------------------------------------------------
template <typename R>
// kind 0: A = M_pc^dag M_pc on even half fields (red-black CGNR);  kind 1: A = M^dag M = H_DW^2 on full fields (unpreconditioned
// CGNR, Table V).  In both A p = O2(O1 p) with <p, A p> = |O1 p|^2.
static int cg_t(dwf_ctx* h, const void* b, void* x, int iters, int nrhs = 1, double tol_rel = 0.0, int check_every = 10, int* done = nullptr,
                int kind = 0) {
    using G = typename Prec<R>::G;
    const size_t hb = half_bytes(h, nrhs) * (kind ? 2 : 1);
    const long long ng = half_groups(h, nrhs) * (kind ? 2 : 1);
    auto op1 = [&](const void* in, void* out, void* tmp, double* norm_out) -> int {
        if (kind == 0) return schur_op(h, false, in, out, tmp, nrhs, norm_out);
        if (int rc = full_op(h, HM_HOP_SELF_G5, false, -0.5, h->mass, in, out, nrhs)) return rc;
        return norm_out ? reduce_to(h, true, out, nullptr, nrhs, 0, norm_out, 1, 1) : DWF_OK;
    };
    auto op2 = [&](const void* in, void* out, void* tmp) -> int {
        if (kind == 0) return schur_op(h, true, in, out, tmp, nrhs);
        return full_op(h, HM_HOP_SELF_G5, false, -0.5, h->mass, in, out, nrhs);
    };
    const int BS = run_groups(h);
    G* r = (G*)h->ws; G* p = (G*)((char*)h->ws + hb); G* w = (G*)((char*)h->ws + 2 * hb);
    G* q = (G*)((char*)h->ws + 3 * hb); void* tmp = (char*)h->ws + 4 * hb;
    double* hist = h->scal; double* pAp = h->scal + (size_t)(iters + 1) * nrhs;     // hist[k*nrhs + r], pAp[k*nrhs + r]
    const unsigned blocks = blas_blocks(h, ng, (long long)BS * nrhs);
    cudaStream_t st = h->stream;
    if (int rc = op1(x, w, tmp, nullptr)) return rc;
    if (int rc = op2(w, q, tmp)) return rc;
    cg_init_kernel<R><<<blocks, 256, 0, st>>>((const G*)b, q, r, p, ng, BS, nrhs, h->partial); LAUNCH_CHECK(h);
    reduce_final_kernel<<<nrhs, 256, 0, st>>>(h->partial, (int)blocks, nrhs, hist, 1, 1); LAUNCH_CHECK(h);
    // Fused iteration (tiled kernel, one rhs, red-black): 5 launches, 15 half-vector passes instead of 8 launches and 19 passes:
    //   w = M p with |w|^2 summed inside K2;  r <- r - alpha M^dag w with |r|^2 summed inside the adjoint K2 (q is never stored);
    //   x += alpha p and p = r + beta p in one pass.
    const bool fusedcg = kind == 0 && norm_fusable(h, nrhs);
    for (int k = 0; k < iters; k++) {
        double* hk = hist + (size_t)k * nrhs; double* hk1 = hk + nrhs; double* pk = pAp + (size_t)k * nrhs;
        if (int rc = op1(p, w, tmp, pk)) return rc;                                // w = O1 p and <p, A p> = |w|^2
        if (fusedcg) {
            const SchurFuse f{r, hk, pk};
            if (int rc = schur_op(h, true, w, nullptr, tmp, nrhs, hk1, &f)) return rc;
            cg_update_xp_kernel<R><<<blocks, 256, 0, st>>>((G*)x, p, r, ng, BS, nrhs, hk, pk, hk1); LAUNCH_CHECK(h);
        } else {
            if (int rc = op2(w, q, tmp)) return rc;
            cg_update_xr_kernel<R><<<blocks, 256, 0, st>>>((G*)x, r, p, q, ng, BS, nrhs, hk, pk, h->partial); LAUNCH_CHECK(h);
            reduce_final_kernel<<<nrhs, 256, 0, st>>>(h->partial, (int)blocks, nrhs, hk1, 1, 1); LAUNCH_CHECK(h);
            cg_update_p_kernel<R><<<blocks, 256, 0, st>>>(p, r, ng, BS, nrhs, hk1, hk); LAUNCH_CHECK(h);
        }
        if (done) *done = k + 1;
        if (tol_rel > 0.0 && ((k + 1) % check_every == 0 || k + 1 == iters)) {      // stopping test (nrhs = 1): |r_k|^2 <= tol^2 |r_0|^2
            CUDA_TRY(h, cudaMemcpyAsync(h->scal_host, hist, sizeof(double), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(h, cudaMemcpyAsync(h->scal_host + 1, hk1, sizeof(double), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(h, cudaStreamSynchronize(st));
            if (h->scal_host[1] <= tol_rel * tol_rel * h->scal_host[0]) break;
        }
    }
    return DWF_OK;
}

static int cg_schur_impl(dwf_handle h, const void* b_even, void* x_even, int iters, int nrhs, double* hist_host, int kind = 0) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS) FAIL(h, DWF_EINVAL, "nrhs must be in [1,%d]", MAX_NRHS);
    if (iters < 0 || 2 * (long long)(iters + 1) * nrhs > SCAL_DOUBLES) FAIL(h, DWF_EINVAL, "iters out of range");
    if (int rc = check_field(h, b_even, "b_even")) return rc;
    if (int rc = check_field(h, x_even, "x_even")) return rc;
    if (b_even == x_even) FAIL(h, DWF_EINVAL, "b == x");
    if (!h->have_gauge) FAIL(h, DWF_ENOGAUGE, "dwf_set_gauge has not been called");
    if (int rc = need_ws(h, (kind ? 8 : 5) * half_bytes(h, nrhs))) return rc;
    // The host loop only enqueues (alpha, beta live on the device).  At launch-bound sizes (a half field of a few MB: configs[1],
    // where an iteration is five kernels of a few microseconds) the whole solve is captured once into a CUDA graph, kept
    // instantiated in the handle, and re-launched as one unit whenever the same (b, x, iters, nrhs, workspace) recur; other
    // arguments re-capture.  DWF_CG_GRAPH=0 / 1 forces it off / on for every size.
    const bool small = half_bytes(h, nrhs) * (kind ? 2 : 1) <= ((size_t)8 << 20);
    const bool use_graph = iters > 0 && (h->cg_graph == 1 || (h->cg_graph < 0 && small));
    int rc;
    if (use_graph) {
        cudaStream_t user = h->stream;
        const bool hit = h->cg_exec && h->cg_b == b_even && h->cg_x == x_even && h->cg_ws == h->ws && h->cg_ws_bytes == h->ws_bytes
                      && h->cg_iters == iters && h->cg_nrhs == nrhs && h->cg_kind == kind;
        if (!hit) {
            if (h->cg_exec) { cudaGraphExecDestroy(h->cg_exec); h->cg_exec = nullptr; }
            cudaGraph_t graph = nullptr;
            CUDA_TRY(h, cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
            h->stream = h->cap_stream;
            const long long launches0 = h->launches;
            rc = h->prec == DWF_F32 ? cg_t<float>(h, b_even, x_even, iters, nrhs, 0.0, 10, nullptr, kind) : cg_t<double>(h, b_even, x_even, iters, nrhs, 0.0, 10, nullptr, kind);
            h->stream = user;
            cudaError_t e = cudaStreamEndCapture(h->cap_stream, &graph);
            if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (e != cudaSuccess) FAIL(h, DWF_ECUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e));
            e = cudaGraphInstantiate(&h->cg_exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) { h->cg_exec = nullptr; FAIL(h, DWF_ECUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e)); }
            h->cg_b = b_even; h->cg_x = x_even; h->cg_ws = h->ws; h->cg_ws_bytes = h->ws_bytes;
            h->cg_iters = iters; h->cg_nrhs = nrhs; h->cg_kind = kind;
            h->cg_launches = h->launches - launches0;
            h->launches = launches0;                           // capture only records: the launches are counted when the graph runs
        }
        CUDA_TRY(h, cudaGraphLaunch(h->cg_exec, user));
        h->launches += h->cg_launches;
    } else {
        rc = h->prec == DWF_F32 ? cg_t<float>(h, b_even, x_even, iters, nrhs, 0.0, 10, nullptr, kind) : cg_t<double>(h, b_even, x_even, iters, nrhs, 0.0, 10, nullptr, kind);
        if (rc) return rc;
    }
    const size_t nh = (size_t)(iters + 1) * nrhs;
    CUDA_TRY(h, cudaMemcpyAsync(h->scal_host, h->scal, nh * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (hist_host) memcpy(hist_host, h->scal_host, nh * sizeof(double));
    return DWF_OK;
}

extern "C" int dwf_cg_schur(dwf_handle h, const void* b_even, void* x_even, int iters, double* hist_host) {
    return cg_schur_impl(h, b_even, x_even, iters, 1, hist_host);
}
extern "C" int dwf_cg_schur_multi(dwf_handle h, const void* b_even, void* x_even, int iters, int nrhs, double* hist_host) {
    return cg_schur_impl(h, b_even, x_even, iters, nrhs, hist_host);
}
extern "C" int dwf_cg_normal(dwf_handle h, const void* b, void* x, int iters, int nrhs, double* hist_host) {
    return cg_schur_impl(h, b, x, iters, nrhs, hist_host, 1);
}

// ------------------------------------------------------------------------------------------------
// BiCGSTAB on the Pauli-Villars preconditioned operator A = M_PV^dag M = D_PV^dag D_DW (PAPER.md L101-107,
// Table V, ref. [31] van der Vorst).  Full native fields, one right-hand side; x holds x_0 on entry.
//   r_0 = b - A x_0, rhat0 = r_0, p_1 = r_0;  per iteration i:
//   rho_i = <rhat0, r_{i-1}>; p_i = r_{i-1} + beta_i (p_{i-1} - omega_{i-1} v_{i-1}); v_i = A p_i; alpha_i = rho_i/<rhat0, v_i>;
//   s = r_{i-1} - alpha_i v_i; t = A s; omega_i = <t,s>/<t,t>; x_i = x_{i-1} + alpha_i p_i + omega_i s; r_i = s - omega_i t.
// The host loop only enqueues: every scalar stays on the device (dwf_aux.cuh, slots of 8 doubles per iteration); 12 launches
// and 2 applies of A (4 stencil launches) per iteration.  Workspace: r(=s), rhat0, p, v, t + the scratch of A = 6 full fields.
// ------------------------------------------------------------------------------------------------
template <typename R>
static int bicgstab_t(dwf_ctx* h, const void* b, void* x, int iters) {
    using G = typename Prec<R>::G;
    const size_t fb = 2 * half_bytes(h, 1);
    const long long ng = 2 * half_groups(h, 1);
    G* r = (G*)h->ws; G* rhat = (G*)((char*)h->ws + fb); G* p = (G*)((char*)h->ws + 2 * fb);
    G* v = (G*)((char*)h->ws + 3 * fb); G* t = (G*)((char*)h->ws + 4 * fb); void* scratch = (char*)h->ws + 5 * fb;
    auto A = [&](const void* in, void* out) -> int {                            // out = D_PV^dag (D_DW in)
        if (int rc = full_op(h, HM_HOP_SELF, false, -0.5, h->mass, in, scratch, 1)) return rc;
        return full_op(h, HM_HOP_SELF, true, -0.5, 1.0, scratch, out, 1);
    };
    const unsigned blocks = (unsigned)std::min<long long>((ng + 255) / 256, (long long)h->sm_count * 8);
    cudaStream_t st = h->stream;
    double* S = h->scal;                                                        // slot(i) = S + 8 i
    if (int rc = A(x, v)) return rc;
    bicg_init_kernel<R><<<blocks, 256, 0, st>>>((const G*)b, v, r, rhat, ng, h->partial); LAUNCH_CHECK(h);
    reduce_final4_kernel<<<1, 256, 0, st>>>(h->partial, (int)blocks, S, 7, -1, 8 + 0, 8 + 1); LAUNCH_CHECK(h);   // |r_0|^2 ; rho_1
    for (int i = 1; i <= iters; i++) {
        double* slot = S + 8 * (size_t)i;
        bicg_p_kernel<R><<<blocks, 256, 0, st>>>(p, r, v, ng, slot - 8, slot, i == 1); LAUNCH_CHECK(h);
        if (int rc = A(p, v)) return rc;
        inner_pair_kernel<R><<<blocks, 256, 0, st>>>(rhat, v, ng, h->partial); LAUNCH_CHECK(h);
        reduce_final4_kernel<<<1, 256, 0, st>>>(h->partial, (int)blocks, slot, 2, 3, -1, -1); LAUNCH_CHECK(h);    // <rhat0, v_i>
        bicg_s_kernel<R><<<blocks, 256, 0, st>>>(r, v, ng, slot); LAUNCH_CHECK(h);
        if (int rc = A(r, t)) return rc;
        inner_pair_kernel<R><<<blocks, 256, 0, st>>>(t, r, ng, h->partial); LAUNCH_CHECK(h);
        reduce_final4_kernel<<<1, 256, 0, st>>>(h->partial, (int)blocks, slot, 4, 5, 6, -1); LAUNCH_CHECK(h);     // <t,s>, <t,t>
        bicg_xr_kernel<R><<<blocks, 256, 0, st>>>((G*)x, r, p, t, rhat, ng, slot, h->partial); LAUNCH_CHECK(h);
        reduce_final4_kernel<<<1, 256, 0, st>>>(h->partial, (int)blocks, slot, 7, -1, 8 + 0, 8 + 1); LAUNCH_CHECK(h);   // |r_i|^2 ; rho_{i+1}
    }
    return DWF_OK;
}

extern "C" int dwf_bicgstab_pv(dwf_handle h, const void* b, void* x, int iters, double* resid2_hist_host) {
    if (!h) return DWF_EINVAL;
    if (iters < 0 || 8 * ((long long)iters + 2) > SCAL_DOUBLES) FAIL(h, DWF_EINVAL, "iters must be in [0,%d]", SCAL_DOUBLES / 8 - 2);
    if (int rc = check_field(h, b, "b")) return rc;
    if (int rc = check_field(h, x, "x")) return rc;
    if (b == x) FAIL(h, DWF_EINVAL, "b == x");
    if (!h->have_gauge) FAIL(h, DWF_ENOGAUGE, "dwf_set_gauge has not been called");
    if (int rc = need_ws(h, 12 * half_bytes(h, 1))) return rc;
    if ((size_t)std::min<long long>((2 * half_groups(h, 1) + 255) / 256, (long long)h->sm_count * 8) * 4 > h->partial_doubles)
        FAIL(h, DWF_EUNSUPPORTED, "reduction scratch too small");
    if (int rc = h->prec == DWF_F32 ? bicgstab_t<float>(h, b, x, iters) : bicgstab_t<double>(h, b, x, iters)) return rc;
    CUDA_TRY(h, cudaMemcpyAsync(h->scal_host, h->scal, 8 * ((size_t)iters + 1) * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (resid2_hist_host) for (int i = 0; i <= iters; i++) resid2_hist_host[i] = h->scal_host[8 * (size_t)i + 7];
    return DWF_OK;
}

// ------------------------------------------------------------------------------------------------
// Complete red-black solve of D_DW psi = eta (Table V, eq. 9), nrhs = 1:
//   eta'_e = eta_e - M_eo M_oo^-1 eta_o ;  CGNR: M_pc^dag M_pc psi_e = M_pc^dag eta'_e (stop: |r_k| <= tol |r_0|, tested
//   every 10 iterations) ;  psi_o = M_oo^-1 (eta_o - M_oe psi_e) ;  M_eo = M_oe = -1/2 Dhop.
// Workspace halves: [0,5) CG, 5: b, 6: t / Schur scratch, 7: hop scratch.  psi_o doubles as scratch until the end.
// ------------------------------------------------------------------------------------------------
extern "C" int dwf_solve(dwf_handle h, const void* eta, void* psi, double tol, int max_iters, int* iters_host, double* relres_host) {
    if (!h) return DWF_EINVAL;
    if (!(tol > 0.0) || max_iters < 1 || 2 * max_iters + 2 > SCAL_DOUBLES) FAIL(h, DWF_EINVAL, "need tol > 0 and 1 <= max_iters <= %d", SCAL_DOUBLES / 2 - 1);
    if (int rc = check_field(h, eta, "eta")) return rc;
    if (int rc = check_field(h, psi, "psi")) return rc;
    if (eta == psi) FAIL(h, DWF_EINVAL, "eta == psi");
    if (!h->have_gauge) FAIL(h, DWF_ENOGAUGE, "dwf_set_gauge has not been called");
    const size_t hb = half_bytes(h, 1);
    if (int rc = need_ws(h, 8 * hb)) return rc;
    const char* eta_e = (const char*)eta; const char* eta_o = eta_e + hb;
    char* psi_e = (char*)psi; char* psi_o = psi_e + hb;
    {                                                         // eta = 0: psi = 0 (CG on a zero right-hand side would divide 0 by 0)
        double ne0 = 0;
        if (int rc = dwf_norm2(h, eta, &ne0, 1, 0)) return rc;
        if (!(ne0 > 0.0)) {
            if (ne0 != 0.0) FAIL(h, DWF_EINVAL, "eta is not finite");
            CUDA_TRY(h, cudaMemsetAsync(psi, 0, 2 * hb, h->stream));
            CUDA_TRY(h, cudaStreamSynchronize(h->stream));
            if (iters_host) *iters_host = 0;
            if (relres_host) *relres_host = 0.0;
            return DWF_OK;
        }
    }
    char* B = (char*)h->ws + 5 * hb; char* T = (char*)h->ws + 6 * hb; char* W = (char*)h->ws + 7 * hb;
    const double half[2] = {0.5, 0.0};
    auto hop_to = [&](int parity_out, const void* in, void* out) -> int {       // out_p = Dhop in_{1-p}
        HopCall k{}; k.mode = HM_HOP; k.dag = false; k.nslots = 1; k.parity0 = parity_out; k.nrhs = 1;
        k.in_hop[0] = in; k.out[0] = out; k.c_hop = 1.0; k.mass = h->mass;
        return launch_hop(h, k);
    };
    // source preparation
    if (int rc = launch_mooinv(h, eta_o, T, 1, h->mass, false)) return rc;
    if (int rc = hop_to(0, T, W)) return rc;
    CUDA_TRY(h, cudaMemcpyAsync(psi_o, eta_e, hb, cudaMemcpyDeviceToDevice, h->stream));
    if (int rc = dwf_axpy(h, half, W, psi_o, 1, 1)) return rc;                   // eta'_e = eta_e + 1/2 Dhop_eo M_oo^-1 eta_o
    if (int rc = schur_op(h, true, psi_o, B, T, 1)) return rc;                   // b = M_pc^dag eta'_e
    // CGNR from x_0 = 0
    CUDA_TRY(h, cudaMemsetAsync(psi_e, 0, hb, h->stream));
    int done = 0;
    int rc = h->prec == DWF_F32 ? cg_t<float>(h, B, psi_e, max_iters, 1, tol, 10, &done) : cg_t<double>(h, B, psi_e, max_iters, 1, tol, 10, &done);
    if (rc) return rc;
    // reconstruction of the odd sites
    if (int rc2 = hop_to(1, psi_e, W)) return rc2;
    CUDA_TRY(h, cudaMemcpyAsync(T, eta_o, hb, cudaMemcpyDeviceToDevice, h->stream));
    if (int rc2 = dwf_axpy(h, half, W, T, 1, 1)) return rc2;                     // eta_o + 1/2 Dhop_oe psi_e
    if (int rc2 = launch_mooinv(h, T, psi_o, 1, h->mass, false)) return rc2;
    // true residual |D_DW psi - eta| / |eta| with the full-lattice operator
    if (relres_host) {
        void* Rf = h->ws;
        if (int rc2 = full_op(h, HM_HOP_SELF, false, -0.5, h->mass, psi, Rf, 1)) return rc2;
        const double minus[2] = {-1.0, 0.0};
        if (int rc2 = dwf_axpy(h, minus, eta, Rf, 1, 0)) return rc2;
        double nr = 0, ne = 0;
        if (int rc2 = dwf_norm2(h, Rf, &nr, 1, 0)) return rc2;
        if (int rc2 = dwf_norm2(h, eta, &ne, 1, 0)) return rc2;
        *relres_host = std::sqrt(nr / ne);
    }
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (iters_host) *iters_host = done;
    return DWF_OK;
}

// ------------------------------------------------------------------------------------------------
// Precision conversion between two handles on the same lattice, and the mixed-precision solve built on it
// ("single and mixed precision").
// ------------------------------------------------------------------------------------------------
extern "C" int dwf_convert(dwf_handle src, dwf_handle dst, const void* in, void* out, int nrhs) {
    if (!src || !dst) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS) FAIL(dst, DWF_EINVAL, "nrhs must be in [1,%d]", MAX_NRHS);
    for (int i = 0; i < 4; i++) if (src->L[i] != dst->L[i]) FAIL(dst, DWF_EINVAL, "dwf_convert: different lattices");
    if (src->Ls != dst->Ls) FAIL(dst, DWF_EINVAL, "dwf_convert: different Ls");
    if (int rc = check_field(dst, in, "in")) return rc;
    if (int rc = check_field(dst, out, "out")) return rc;
    cudaStream_t st = dst->stream;
    if (!src->inv_lex) {
        CUDA_TRY(dst, cudaMalloc((void**)&src->inv_lex, (size_t)src->V4 * sizeof(int)));
        invert_lex_kernel<<<(unsigned)((2 * src->V4h + 255) / 256), 256, 0, st>>>(src->lex, src->inv_lex, src->V4h);
        LAUNCH_CHECK(dst);
    }
    const long long total = 2 * src->V4h * nrhs * 12 * (src->Ls / 2);
    const unsigned blocks = (unsigned)((total + 255) / 256);
#define CONV(RS, RD) convert_kernel<RS, RD><<<blocks, 256, 0, st>>>((const Prec<RS>::G*)in, (Prec<RD>::G*)out, src->inv_lex, dst->lex, \
                                                                    src->V4h, src->Ls, nrhs, src->sg_shift, dst->sg_shift, 2)
    if (src->prec == DWF_F64 && dst->prec == DWF_F32) CONV(double, float);
    else if (src->prec == DWF_F32 && dst->prec == DWF_F64) CONV(float, double);
    else if (src->prec == DWF_F32) CONV(float, float);
    else CONV(double, double);
#undef CONV
    LAUNCH_CHECK(dst);
    return DWF_OK;
}

// D_DW psi = eta to fp64 accuracy with the work done in fp32: defect correction
//   r = eta - D psi (fp64);  e = dwf_solve(h32, r, inner_tol) (fp32 red-black CGNR);  psi += e (fp64);  until |r| <= tol |eta|.
// Both handles: same lattice, Ls, M5, mass, gauge set (the fp32 one with the fp64 links rounded once), workspaces set
// (dwf_workspace_bytes(h, 1) each), same stream.
extern "C" int dwf_solve_mixed(dwf_handle h64, dwf_handle h32, const void* eta, void* psi, double tol, double inner_tol,
                               int max_outer, int max_inner, int* outer_host, int* inner_total_host, double* relres_host) {
    if (!h64 || !h32) return DWF_EINVAL;
    if (h64->prec != DWF_F64 || h32->prec != DWF_F32) FAIL(h64, DWF_EINVAL, "dwf_solve_mixed needs an fp64 and an fp32 handle");
    if (!(tol > 0.0) || !(inner_tol > 0.0) || max_outer < 1 || max_inner < 1) FAIL(h64, DWF_EINVAL, "bad tolerances / iteration limits");
    if (h64->M5 != h32->M5 || h64->mass != h32->mass) FAIL(h64, DWF_EINVAL, "the two handles differ in M5 or mass");
    if (int rc = check_field(h64, eta, "eta")) return rc;
    if (int rc = check_field(h64, psi, "psi")) return rc;
    if (eta == psi) FAIL(h64, DWF_EINVAL, "eta == psi");
    if (!h64->have_gauge || !h32->have_gauge) FAIL(h64, DWF_ENOGAUGE, "dwf_set_gauge has not been called on both handles");
    const size_t hb64 = half_bytes(h64, 1), hb32 = half_bytes(h32, 1);
    if (int rc = need_ws(h64, 6 * hb64)) return rc;
    if (need_ws(h32, 12 * hb32)) FAIL(h64, DWF_ENOWORKSPACE, "fp32 handle: workspace of %zu bytes needed", 12 * hb32);
    char* Dpsi = (char*)h64->ws; char* r64 = Dpsi + 2 * hb64; char* e64 = Dpsi + 4 * hb64;
    char* r32 = (char*)h32->ws + 8 * hb32; char* e32 = (char*)h32->ws + 10 * hb32;
    const double one[2] = {1.0, 0.0}, minus[2] = {-1.0, 0.0};
    double neta = 0, nr = 0;
    if (int rc = dwf_norm2(h64, eta, &neta, 1, 0)) return rc;
    if (!(neta > 0.0)) FAIL(h64, DWF_EINVAL, "eta is zero");
    CUDA_TRY(h64, cudaMemsetAsync(psi, 0, 2 * hb64, h64->stream));
    int outer = 0, inner_total = 0;
    double rel = 1.0;
    for (;;) {
        // r = eta - D psi
        if (outer == 0) CUDA_TRY(h64, cudaMemcpyAsync(r64, eta, 2 * hb64, cudaMemcpyDeviceToDevice, h64->stream));
        else {
            if (int rc = full_op(h64, HM_HOP_SELF, false, -0.5, h64->mass, psi, Dpsi, 1)) return rc;
            CUDA_TRY(h64, cudaMemcpyAsync(r64, eta, 2 * hb64, cudaMemcpyDeviceToDevice, h64->stream));
            if (int rc = dwf_axpy(h64, minus, Dpsi, r64, 1, 0)) return rc;
        }
        if (int rc = dwf_norm2(h64, r64, &nr, 1, 0)) return rc;
        rel = std::sqrt(nr / neta);
        if (rel <= tol || outer == max_outer) break;
        // inner solve in fp32 on the residual (floating point: its relative accuracy does not depend on the size of r)
        if (int rc = dwf_convert(h64, h32, r64, r32, 1)) return rc;
        int it = 0;
        if (int rc = dwf_solve(h32, r32, e32, inner_tol, max_inner, &it, nullptr)) { snprintf(h64->err, sizeof(h64->err), "inner solve: %.200s", h32->err); return rc; }
        inner_total += it;
        if (int rc = dwf_convert(h32, h64, e32, e64, 1)) return rc;
        if (int rc = dwf_axpy(h64, one, e64, psi, 1, 0)) return rc;
        outer++;
    }
    CUDA_TRY(h64, cudaStreamSynchronize(h64->stream));
    if (outer_host) *outer_host = outer;
    if (inner_total_host) *inner_total_host = inner_total;
    if (relres_host) *relres_host = rel;
    return DWF_OK;
}

// ------------------------------------------------------------------------------------------------
// End-to-end apply from host canonical arrays (bench.py's e2e leg): H2D, import, apply, export, D2H.
// Workspace use: [0, F) canonical staging / native out, [F, 2F) native in / canonical out, [2F, ...) the operator's own scratch
// (SCHUR_EO: 1 half field, SCHUR_EO_ALT and MPVDAG_M: 2)
// ------------------------------------------------------------------------------------------------
// dwf_apply_host for the one-launch full-lattice operators, pipelined over chunks of t-slices: while chunk c is converted and
// applied, chunk c+1 arrives over PCIe and chunk c-1 leaves (the two copy directions run at the same time).  The canonical
// layout [rhs][s][t][...] makes a t-range one 2-D copy (rows = (rhs, s)); in the native order (lexicographic blocks, t slowest) it
// is a contiguous range of sites and of work items.  A chunk's operator needs its two t-neighbour chunks imported.
// Buffers: A = canonical in, then canonical out chunk by chunk; B = native in; C = native out (6 half fields).
static int apply_host_pipelined(dwf_ctx* h, int mode, bool dag, double c_hop, double mass, const void* in_host, void* out_host, int nrhs, int nc) {
    const size_t hb = half_bytes(h, nrhs), fb = 2 * hb, R = real_bytes(h);
    char* A = (char*)h->ws; char* B = A + fb; char* C = B + fb;
    if (!h->io_in) {
        CUDA_TRY(h, cudaStreamCreateWithFlags(&h->io_in, cudaStreamNonBlocking));
        CUDA_TRY(h, cudaStreamCreateWithFlags(&h->io_out, cudaStreamNonBlocking));
        for (cudaEvent_t& e : h->io_ev) CUDA_TRY(h, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    cudaEvent_t* ev_in = h->io_ev; cudaEvent_t* ev_out = h->io_ev + 16; cudaEvent_t ev_start = h->io_ev[32];
    const int Lt = h->L[3], tc = Lt / nc;                                        // t-slices per chunk
    const size_t slice = (size_t)h->V4 / Lt * 24 * R;                           // one t-slice of one (rhs, s) row
    const size_t pitch = slice * Lt, width = slice * tc;
    const size_t rows = (size_t)nrhs * h->Ls;
    const long long sc = h->V4h / nc;                                            // sites per parity per chunk
    cudaStream_t st = h->stream;
    CUDA_TRY(h, cudaEventRecord(ev_start, st));                                  // earlier work on the handle's stream may still use the workspace
    CUDA_TRY(h, cudaStreamWaitEvent(h->io_in, ev_start, 0));
    CUDA_TRY(h, cudaStreamWaitEvent(h->io_out, ev_start, 0));
    for (int c = 0; c < nc; c++) {
        CUDA_TRY(h, cudaMemcpy2DAsync(A + c * width, pitch, (const char*)in_host + c * width, pitch, width, rows, cudaMemcpyHostToDevice, h->io_in));
        CUDA_TRY(h, cudaEventRecord(ev_in[c], h->io_in));
    }
    auto run_chunk = [&](int c) -> int {                                         // operator, export and D2H of chunk c
        if (int rc = full_op(h, mode, dag, c_hop, mass, B, C, nrhs, 0, nullptr, 0, nullptr, 0, c * sc, (c + 1) * sc)) return rc;
        const int rc = h->prec == DWF_F32 ? reorder_spinor<float, false>(h, nullptr, A, C, nrhs, -1, c * sc, (c + 1) * sc)
                                          : reorder_spinor<double, false>(h, nullptr, A, C, nrhs, -1, c * sc, (c + 1) * sc);
        if (rc) return rc;
        CUDA_TRY(h, cudaEventRecord(ev_out[c], st));
        CUDA_TRY(h, cudaStreamWaitEvent(h->io_out, ev_out[c], 0));
        CUDA_TRY(h, cudaMemcpy2DAsync((char*)out_host + c * width, pitch, A + c * width, pitch, width, rows, cudaMemcpyDeviceToHost, h->io_out));
        return DWF_OK;
    };
    for (int c = 0; c < nc; c++) {
        CUDA_TRY(h, cudaStreamWaitEvent(st, ev_in[c], 0));
        const int rc = h->prec == DWF_F32 ? reorder_spinor<float, true>(h, A, nullptr, B, nrhs, -1, c * sc, (c + 1) * sc)
                                          : reorder_spinor<double, true>(h, A, nullptr, B, nrhs, -1, c * sc, (c + 1) * sc);
        if (rc) return rc;
        if (c >= 2) { if (int rc2 = run_chunk(c - 1)) return rc2; }              // chunks c-2, c-1, c are in
    }
    if (int rc = run_chunk(nc - 1)) return rc;                                   // periodic in t: the last and the first chunk need each other
    if (int rc = run_chunk(0)) return rc;
    CUDA_TRY(h, cudaStreamSynchronize(h->io_out));
    CUDA_TRY(h, cudaStreamSynchronize(st));
    return DWF_OK;
}

extern "C" int dwf_apply_host(dwf_handle h, int op, const void* in_host, void* out_host, int nrhs) {
    if (!h) return DWF_EINVAL;
    if (nrhs < 1 || nrhs > MAX_NRHS) FAIL(h, DWF_EINVAL, "nrhs must be in [1,%d]", MAX_NRHS);
    if (!in_host || !out_host) FAIL(h, DWF_EINVAL, "NULL host pointer");
    const int base = op & ~DWF_DAGGER;
    const bool halfop = (base == DWF_SCHUR_EO || base == DWF_MEE || base == DWF_MOOINV || base == DWF_SCHUR_EO_ALT);
    if (base != DWF_MEE && base != DWF_MOOINV && !h->have_gauge) FAIL(h, DWF_ENOGAUGE, "dwf_set_gauge has not been called");
    const size_t hb = half_bytes(h, nrhs), fb = 2 * hb;
    // One-launch full-lattice operators with 6 half fields of workspace: copies pipelined against the kernels in chunks of t-slices
    // (at least 3 chunks of whole block layers, at most 16).  Everything else: the serial path below.
    if ((base == DWF_DHOP || base == DWF_DDW || base == DWF_DPV || base == DWF_HDW) && h->blk_t > 0 && h->ws
        && h->ws_bytes >= 3 * fb && in_host != out_host && !getenv("DWF_NO_HOST_PIPELINE")) {
        const int layers = h->L[3] / h->blk_t;
        int nc = 0;
        for (int n = std::min(layers, 16); n >= 3; n--) if (layers % n == 0) { nc = n; break; }
        if (nc && (h->V4h / nc) % partial_unit(h) == 0) {
            const bool dag = (op & DWF_DAGGER) != 0;
            switch (base) {
                case DWF_DHOP: return apply_host_pipelined(h, HM_HOP, dag, 1.0, h->mass, in_host, out_host, nrhs, nc);
                case DWF_DDW:  return apply_host_pipelined(h, HM_HOP_SELF, dag, -0.5, h->mass, in_host, out_host, nrhs, nc);
                case DWF_DPV:  return apply_host_pipelined(h, HM_HOP_SELF, dag, -0.5, 1.0, in_host, out_host, nrhs, nc);
                default:       return apply_host_pipelined(h, HM_HOP_SELF_G5, false, -0.5, h->mass, in_host, out_host, nrhs, nc);
            }
        }
    }
    // scratch of the operator itself, behind the two staging fields
    const size_t op_ws = (base == DWF_SCHUR_EO) ? hb : (base == DWF_SCHUR_EO_ALT || base == DWF_MPVDAG_M) ? 2 * hb : 0;
    if (int rc = need_ws(h, 2 * fb + op_ws)) return rc;
    char* A = (char*)h->ws; char* B = A + fb; void* tmp = A + 2 * fb;
    void* saved_ws = h->ws; size_t saved_n = h->ws_bytes;
    CUDA_TRY(h, cudaMemcpyAsync(A, in_host, fb, cudaMemcpyHostToDevice, h->stream));
    // full ops: native in = B, native out = A (canonical staging is dead after import), canonical out = B
    // half ops: native in = B[0,hb), native out = B[hb,2hb), canonical out = A (zeroed: odd sites read 0)
    void* nat_in = B; void* nat_out = halfop ? (void*)(B + hb) : (void*)A; void* can_out = halfop ? (void*)A : (void*)B;
    int rc = dwf_import(h, A, nat_in, nrhs, halfop ? 0 : -1);
    if (!rc) {
        h->ws = tmp; h->ws_bytes = op_ws;              // the operator's scratch lives behind the two staging buffers
        rc = apply_checked(h, op, nat_in, nat_out, nrhs);
        h->ws = saved_ws; h->ws_bytes = saved_n;
    }
    if (rc) return rc;
    if (halfop) CUDA_TRY(h, cudaMemsetAsync(can_out, 0, fb, h->stream));
    rc = dwf_export(h, nat_out, can_out, nrhs, halfop ? 0 : -1);
    if (rc) return rc;
    CUDA_TRY(h, cudaMemcpyAsync(out_host, can_out, fb, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return DWF_OK;
}
