/*
 * dwf.h -- C ABI of libdwf: the data-parallel hot path of arxiv 2103.05034 (Boyle & Yamaguchi,
 * "Comparison of Domain Wall Fermion Multigrid Methods") as hand-written CUDA for sm_100a (B200).
 *
 * What is computed (PAPER.md = /root/reference/PAPER.md line numbers; readings R1..R22 = DESIGN.md sec. 2):
 *   D_hop      eq. 2  L30   Wilson hopping stencil, spin-projected, SU(3) links
 *   D_DW       eq. 4  L39 + eq. 5 L43   5D Shamir domain-wall operator
 *   H_DW       eq. 6  L48   Gamma5 D_DW, Gamma5 = gamma5 R5 (L46)
 *   D_PV       L50          D_DW at unit mass
 *   M_pc       Table V L386 even-odd Schur operator M_ee - M_eo M_oo^{-1} M_oe (acts on EVEN half fields)
 *   Chebyshev  eq. 23, map L173, eq. 34 L227   T_order(2(H_DW^2 - lo)/(hi - lo) - 1)
 *   rb-CGNR    eq. 9  L73   CG on M_pc^dag M_pc
 * Conventions: chiral gamma basis (R1), P+- = (1 +- gamma5)/2 (R2), periodic in x,y,z and
 * antiperiodic in t (R3), 4D red-black parity (x+y+z+t)&1 with even = 0 (R8).
 *
 * Pointers: every `const void* / void*` FIELD argument is a DEVICE pointer, 16-byte aligned, owned
 * by the caller (e.g. a torch tensor's data_ptr); the library never frees or retains it beyond the
 * call (work is enqueued on the handle's stream; the buffer must stay alive until that work is
 * done).  Pointers named *_host are HOST pointers.  The handle owns only its gauge copy, its
 * index tables and a few KB of reduction scratch (cudaMalloc at dwf_create / dwf_set_gauge).
 *
 * Layouts.
 *   canonical spinor : complex<real> [nrhs][Ls][t][z][y][x][spin 4][colour 3], re/im interleaved
 *   canonical gauge  : complex<real> [mu 4][t][z][y][x][a 3][b 3], mu = 0..3 <-> x,y,z,t,
 *                      (U psi)_a = sum_b U_ab psi_b
 *   native spinor    : opaque; dwf_field_bytes() gives its size; a full field is
 *                      the even half field followed by the odd half field; convert with
 *                      dwf_import / dwf_export.  `real` is float (DWF_F32) or double (DWF_F64).
 *
 * Errors: every int-returning call returns DWF_OK or a negative code and never throws or exits;
 * dwf_last_error() gives a message.  Calls are asynchronous on the handle's stream unless they
 * return host values (dwf_inner, dwf_norm2, dwf_cg_schur, dwf_apply_host: these synchronise).
 * One handle per host thread.
 */
#ifndef DWF_H
#define DWF_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dwf_ctx* dwf_handle;

enum { DWF_F32 = 0, DWF_F64 = 1 };

/* Operators for dwf_apply.  Full-field ops: DHOP, DDW, HDW, DPV.  Half-field ops: SCHUR_EO (even
 * in, even out), MEE (M_ee = M_oo: the 4D-site-diagonal part 5-M5 + fifth-dimension hops of eq. 4)
 * and MOOINV (its exact inverse, closed form of DESIGN.md sec. 5.4).
 * OR-ing DWF_DAGGER applies the adjoint (valid for every op; H_DW is hermitian so it is a no-op). */
enum { DWF_DHOP = 0, DWF_DDW = 1, DWF_HDW = 2, DWF_DPV = 3, DWF_SCHUR_EO = 4, DWF_MEE = 5, DWF_MOOINV = 6,
       DWF_MPVDAG_M = 7,   /* Pauli-Villars preconditioned operator D_PV^dag D_DW; full fields; uses the
                              workspace (1 full field); with DWF_DAGGER: D_DW^dag D_PV */
       DWF_SCHUR_EO_ALT = 8, /* the other Schur form of Table V (L387): 1 - M_ee^-1 M_eo M_oo^-1 M_oe on EVEN half fields;
                              uses the workspace (2 half fields); with DWF_DAGGER its adjoint */
       DWF_DAGGER = 0x100 };

enum { DWF_OK = 0, DWF_EINVAL = -1, DWF_ENOGAUGE = -2, DWF_ENOMEM = -3, DWF_ECUDA = -4,
       DWF_EUNSUPPORTED = -5, DWF_ENOWORKSPACE = -6,
       DWF_ERANGE = -7 /* a result left the range of the field's precision (dwf_chebyshev_subspace) */ };

/* Create a handle.  L = {Lx,Ly,Lz,Lt}, each even and >= 4; Ls even, 2 <= Ls <= 64 (closed-form M_oo^{-1}
 * is instantiated for Ls in {4,8,12,16,24,32}: other Ls -> DWF_EUNSUPPORTED from SCHUR_EO/MOOINV/CG).
 * M5 = domain-wall height (eq. 5), mass = m of eq. 4.  M5 == 5 or 1 + m (5-M5)^-Ls == 0 -> DWF_EINVAL
 * (M_oo singular).  precision: DWF_F32 / DWF_F64 = storage and arithmetic type of fields and links;
 * reductions always accumulate in fp64.  Uses the current CUDA device. */
int dwf_create(const int L[4], int Ls, double M5, double mass, int precision, dwf_handle* out);
int dwf_destroy(dwf_handle h);

/* Stream on which all later work of this handle is enqueued (a cudaStream_t; NULL = default). */
int dwf_set_stream(dwf_handle h, void* cuda_stream);

/* Scratch.  The library never allocates field memory: the caller provides a device buffer and keeps it alive while
 * the handle uses it.  dwf_workspace_bytes(h, nrhs) is enough for EVERY call with up to nrhs right-hand sides
 * (12 half fields + 256 bytes); a caller that makes only some calls may register less -- each call below states
 * its need in half fields of nrhs right-hand sides (dwf_field_bytes(h, nrhs, 1)) and returns DWF_ENOWORKSPACE if
 * the registered buffer is smaller: SCHUR_EO 1, SCHUR_EO_ALT 2, MPVDAG_M 2, dwf_chebyshev 4, dwf_chebyshev_subspace 6,
 * dwf_chebyshev_smoother 8, dwf_power_lambda_max 4, dwf_cg_schur(_multi) 5, dwf_cg_normal 8, dwf_bicgstab_pv 12, dwf_apply_host 4 + the
 * operator's own need, dwf_solve 8,
 * dwf_solve_mixed 6 (fp64 handle) + 12 (fp32 handle). */
size_t dwf_workspace_bytes(dwf_handle h, int nrhs);
int dwf_set_workspace(dwf_handle h, void* dev_ptr, size_t nbytes);

/* Copy + reorder a canonical gauge field (device pointer, handle precision) into the handle.
 * The antiperiodic-t sign is folded into the stored U_t on the last time slice.  Stream-ordered. */
int dwf_set_gauge(dwf_handle h, const void* U_canonical_dev);

/* Bytes of a native field of nrhs right-hand sides; half = 0: full lattice, 1: one parity. */
size_t dwf_field_bytes(dwf_handle h, int nrhs, int half);

/* canonical (device) <-> native (device).  parity = -1: full field; 0 / 1: the canonical array is a
 * full-lattice array, only sites of that parity are read (import) / written (export; the other
 * sites are left untouched), the native buffer is a half field. */
int dwf_import(dwf_handle h, const void* canonical_dev, void* native_dev, int nrhs, int parity);
int dwf_export(dwf_handle h, const void* native_dev, void* canonical_dev, int nrhs, int parity);

/* out = OP in, native layout, nrhs fields at once (1 <= nrhs <= 64); in != out. */
int dwf_apply(dwf_handle h, int op, const void* in, void* out, int nrhs);

/* Same operator (every op of dwf_apply, DWF_DAGGER included), end to end from HOST canonical arrays: H2D copy, import,
 * apply, export, D2H copy (synchronises).  Workspace: 4 half fields of staging + the operator's own need.  With 6 half fields the
 * one-launch full-lattice operators (DHOP, DDW, DPV, HDW) run pipelined over chunks of t-slices (host -> device copy of chunk c+1,
 * kernels of chunk c and device -> host copy of chunk c-1 at the same time; in_host != out_host; lattices with at least three
 * t-layers of blocks), which roughly halves the time of a PCIe-bound call; DWF_NO_HOST_PIPELINE=1 keeps the serial path.  For the
 * half-field ops SCHUR_EO/SCHUR_EO_ALT/MEE/MOOINV the arrays are full-lattice canonical arrays of which only the even
 * sites are read; the odd sites of out_host are written as zero. */
int dwf_apply_host(dwf_handle h, int op, const void* in_host, void* out_host, int nrhs);

/* out = T_order(2 (H_DW^2 - lo) / (hi - lo) - 1) in   (eq. 23, eq. 34; R10, R13, R14).
 * order >= 0, hi > lo.  Full native fields; in != out; uses the workspace (2 full fields). */
int dwf_chebyshev(dwf_handle h, int order, double lo, double hi, const void* in, void* out, int nrhs);

/* Subspace generation by Chebyshev filtering of a noise vector (eq. 34-37; setup option 3).
 *   v     = T_m(2 (H_DW^2 - lambda_lo) / (lambda_max - lambda_lo) - 1) eta        first-pass filter, eq. 34 (R10)
 *   phi_k = T_{k delta}(2 H_DW^2 / lambda_max - 1) v ,  k = 0 .. nvec-1            eq. 35, 37 (phi_0 = v, R23)
 * All phi_k come from ONE three-term recurrence started at v ("all for the cost of the highest order", L229):
 * 2 m + 2 (nvec-1) delta operator applies.  phi = nvec consecutive full native fields of nrhs right-hand sides
 * each (phi_k at byte offset k * dwf_field_bytes(h, nrhs, 0)); eta != phi; m >= 0, delta >= 1, nvec >= 1,
 * 0 <= lambda_lo < lambda_max.  No normalisation (R14): outside [lambda_lo, lambda_max] T_m grows as cosh(m acosh|x|),
 * so |phi_0|^2 and |phi_{nvec-1}|^2 are checked and DWF_ERANGE is returned when the precision of the handle overflowed
 * (use an fp64 handle for m, lambda_lo with larger growth).  Uses the workspace (3 full fields).  Synchronises. */
int dwf_chebyshev_subspace(dwf_handle h, int m, double lambda_lo, double lambda_max, int delta, int nvec,
                           const void* eta, void* phi, int nrhs);

/* Chebyshev smoother of degree N on the normal residual system (eq. 24-25):
 *   out = [ c_0/2 + sum_{j=1..N} c_j T_j(2 (M^dag M - a)/(b - a) - 1) ] M^dag r ,  M = D_DW (M^dag M = H_DW^2),
 *   c_j = (2/N) sum_{k=0..N-1} f(y(cos theta_k)) cos(j theta_k), f(y) = 1/y, theta_k = pi (k + 1/2)/N,
 *   y(x) = ((b - a) x + b + a)/2  (the inverse of the interval map of L173): a polynomial approximation of M^-1 on
 *   the part of the spectrum of M^dag M inside [a, b].  1 <= N <= 4096, 0 < a < b; r != out; full native fields.
 * Uses the workspace (4 full fields). */
int dwf_chebyshev_smoother(dwf_handle h, int N, double a, double b, const void* r, void* out, int nrhs);

/* lambda_max(H_DW^2) by the power method (L225; reading R24), nrhs = 1, full native field v (start vector in,
 * last iterate out).  Iteration i: u = H v, lambda_i = |u|^2 / |v|^2 (Rayleigh quotient of H^2),
 * v <- H u / lambda_i.  *lambda_host = lambda_iters; lambda_hist_host (may be NULL) receives all `iters`
 * quotients.  Uses the workspace (2 full fields).  Synchronises. */
int dwf_power_lambda_max(dwf_handle h, int iters, void* v, double* lambda_host, double* lambda_hist_host);

/* BLAS-1 on native fields (half = 0 full, 1 half field), one scalar per right-hand side.
 *   axpy : y <- a x + y, a_host[2*nrhs] = (re, im) per rhs
 *   inner: out_host[2*nrhs] = sum conj(x) y per rhs (fp64 accumulation, deterministic order)
 *   norm2: out_host[nrhs]   = sum |x|^2 per rhs */
int dwf_axpy(dwf_handle h, const double* a_host, const void* x, void* y, int nrhs, int half);
int dwf_inner(dwf_handle h, const void* x, const void* y, double* out_host, int nrhs, int half);
int dwf_norm2(dwf_handle h, const void* x, double* out_host, int nrhs, int half);

/* norm2 for callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the same
 * kernels and summation order as dwf_norm2 (north_star item (4)), but nothing on its path calls cudaMalloc/cudaFree -- the
 * per-block partials live in a file-scope __device__ array of 32768 doubles (256 KB per GPU that loads the library, held until
 * the process exits) -- and out_dev[nrhs] is a DEVICE pointer: the call is asynchronous on the handle's stream.  The handle's
 * device must be the current device.  Sizes whose partials exceed the array (blocks x nrhs x 2 doubles; blocks <= 8 per SM)
 * return DWF_EUNSUPPORTED: use fewer right-hand sides per call.  All calls on a GPU share the array: calls that overlap on the
 * GPU (other streams or handles) race; successive calls on one stream do not (every slot a call reads it has written first). */
int dwf_norm2_static(dwf_handle h, const void* x, double* out_dev, int nrhs, int half);

/* `iters` iterations of Hestenes-Stiefel CG on M_pc^dag M_pc x = b (eq. 9), nrhs = 1, even half
 * fields.  x_even holds x_0 on entry and x_iters on return.  resid2_hist_host (may be NULL) receives
 * iters+1 values |r_k|^2.  Uses the workspace (5 half fields).  Synchronises at the end only.  At launch-bound sizes (a half field
 * of at most 8 MB) the solve is captured into a CUDA graph that the handle keeps and re-launches while (b, x, iters, workspace) recur. */
int dwf_cg_schur(dwf_handle h, const void* b_even, void* x_even, int iters, double* resid2_hist_host);

/* The same CG on nrhs right-hand sides in lock step (one independent CG per rhs: per-rhs alpha, beta; every kernel serves all
 * of them).  b_even, x_even: even half fields of nrhs right-hand sides; resid2_hist_host (may be NULL): (iters+1) * nrhs
 * values, [k][r] = |r_k|^2 of rhs r.  Uses the workspace (5 half fields of nrhs right-hand sides). */
int dwf_cg_schur_multi(dwf_handle h, const void* b_even, void* x_even, int iters, int nrhs, double* resid2_hist_host);

/* Unpreconditioned CGNR (Table V, eq. 9): `iters` iterations of the same CG on M^dag M x = b with M = D_DW
 * (M^dag M = H_DW^2, eq. 11), FULL native fields of nrhs right-hand sides, x holds x_0 on entry.  History as in
 * dwf_cg_schur_multi.  Uses the workspace (8 half fields of nrhs right-hand sides). */
int dwf_cg_normal(dwf_handle h, const void* b, void* x, int iters, int nrhs, double* resid2_hist_host);

/* BiCGSTAB (van der Vorst, PAPER.md ref. [31]) on the Pauli-Villars preconditioned system D_PV^dag D_DW x = b (PAPER.md
 * L101-107; Table V), `iters` iterations, FULL native fields, nrhs = 1; x holds x_0 on entry and x_iters on return.
 * resid2_hist_host (may be NULL) receives iters+1 values |r_i|^2 of the recursive residual r_i of this system.
 * Complex <a,b> = sum conj(a) b; a vanishing denominator (zero right-hand side) freezes the iteration instead of dividing.
 * Uses the workspace (12 half fields).  Enqueue-only (all scalars stay on the device); synchronises at the end. */
int dwf_bicgstab_pv(dwf_handle h, const void* b, void* x, int iters, double* resid2_hist_host);

/* Complete red-black solve of D_DW psi = eta (Table V; eq. 9), nrhs = 1, full native fields:
 *   eta'_e = eta_e - M_eo M_oo^-1 eta_o;  CGNR on M_pc^dag M_pc psi_e = M_pc^dag eta'_e from psi_e = 0, stopped when
 *   |r_k| <= tol |r_0| (r = residual of the normal equations; tested every 10 iterations) or after max_iters;
 *   psi_o = M_oo^-1 (eta_o - M_oe psi_e).
 * *iters_host = CG iterations done; *relres_host (may be NULL) = |D_DW psi - eta| / |eta| recomputed with the
 * full-lattice operator.  eta != psi.  Uses the workspace (8 half fields).  Synchronises. */
int dwf_solve(dwf_handle h, const void* eta, void* psi, double tol, int max_iters, int* iters_host, double* relres_host);

/* Convert a full native field of nrhs right-hand sides from the precision (and site order) of handle `src` to that of
 * handle `dst`: same lattice and Ls.  Enqueued on dst's stream. */
int dwf_convert(dwf_handle src, dwf_handle dst, const void* in_native_src, void* out_native_dst, int nrhs);

/* Mixed-precision solve of D_DW psi = eta ("single and mixed precision"; the usual defect correction):
 *   repeat: r = eta - D_DW psi in fp64 (h64); stop when |r| <= tol |eta| or after max_outer corrections;
 *           e = dwf_solve(h32, r, inner_tol, max_inner) in fp32; psi += e in fp64.
 * h64 / h32: an fp64 and an fp32 handle with the same lattice, Ls, M5, mass, both with gauge and workspace
 * (dwf_workspace_bytes(h, 1)) set and on the same stream.  eta, psi: fp64 full native fields of h64, nrhs = 1.
 * *outer_host = corrections done, *inner_total_host = fp32 CG iterations in total, *relres_host = final |r|/|eta| (fp64). */
int dwf_solve_mixed(dwf_handle h64, dwf_handle h32, const void* eta, void* psi, double tol, double inner_tol,
                    int max_outer, int max_inner, int* outer_host, int* inner_total_host, double* relres_host);

/* Number of kernel launches this handle has enqueued so far (for bench.py's gpu_launches). */
long long dwf_launch_count(dwf_handle h);

/* Message of the last error on this handle (static storage, valid until the next call). */
const char* dwf_last_error(dwf_handle h);

#ifdef __cplusplus
}
#endif
#endif /* DWF_H */
