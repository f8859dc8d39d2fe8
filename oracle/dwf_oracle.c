/*
 * dwf_oracle.c -- CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).
 *
 * A plain, slow, obviously-correct restatement of the operators of arxiv 2103.05034
 * ("Comparison of Domain Wall Fermion Multigrid Methods", PAPER.md) in C99 `double complex`.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * load this library.  It shares NO code with the CUDA path (paper_2103_05034_b200/csrc) and
 * deliberately uses none of its ideas:
 *   - gamma matrices are full 4x4 complex matrices applied as matrix-vector products
 *     (no spin projection to half spinors),
 *   - fields are full-lattice canonical arrays (no checkerboarded storage),
 *   - the antiperiodic-t sign is applied on the hop (not folded into the links),
 *   - adjoints are TRUE adjoints: every non-zero block B(row,col) of the forward operator is
 *     applied as out[col] += B^dagger in[row]  (not via Gamma5 or a swapped projector),
 *   - M_oo^{-1} is a generic dense Gaussian elimination of the Ls x Ls s-matrix per site
 *     (not the closed form the CUDA path uses).
 *
 * Canonical layout (DESIGN.md sec. 3 / SURVEY App. A.1), all complex128, C order:
 *   spinor psi[rhs][s][t][z][y][x][spin 4][colour 3]
 *   gauge  U  [mu 4][t][z][y][x][a 3][b 3]     mu=0..3 <-> x,y,z,t ; (U psi)_a = sum_b U_ab psi_b
 *
 * Passages followed (PAPER.md line numbers):
 *   eq. 1  L25  D_W(M)   = M + 4 - 1/2 D_hop
 *   eq. 2  L30  D_hop    = (1-g_mu) U_mu(x) d_{x+mu,y} + (1+g_mu) U_mu^dag(y) d_{x-mu,y}
 *   eq. 4  L39  D_DW     : s-matrix with D_par on the diagonal, -P_- above, -P_+ below,
 *                          +m P_+ in the (0,Ls-1) corner, +m P_- in the (Ls-1,0) corner
 *   eq. 5  L43  D_par    = 5 - M5 - 1/2 D_hop
 *   L46, eq. 6 L48       Gamma5 = gamma5 R5,  H_DW = Gamma5 D_DW
 *   L50                  D_PV = D_DW at unit mass
 *   Table V L386         M_pc = M_ee - M_eo M_oo^{-1} M_oe  (4D parity, even = 0)
 *   eq. 9  L73           CGNR on M_pc^dag M_pc (Hestenes-Stiefel CG, ref [29])
 *   eq. 23, eq. 34 L227   Chebyshev T_n of the mapped squared operator
 * Readings of what the paper leaves open (gamma basis, P+-, boundary conditions ...) are
 * DESIGN.md sec. 2 R1..R22.  Every function here is pinned by tests/test_oracle_*.py.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>

typedef double complex cplx;

/* ---- R1: chiral gamma basis, gamma_k = [[0,-i sigma_k],[i sigma_k,0]], gamma_t = [[0,1],[1,0]],
 *      gamma5 = gamma_x gamma_y gamma_z gamma_t = diag(1,1,-1,-1).  Index [mu][row][col].   ---- */
static const cplx GAMMA[4][4][4] = {
    { {0, 0, 0, -I}, {0, 0, -I, 0}, {0, I, 0, 0}, {I, 0, 0, 0} },   /* gamma_x */
    { {0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0} },   /* gamma_y */
    { {0, 0, -I, 0}, {0, 0, 0, I}, {I, 0, 0, 0}, {0, -I, 0, 0} },   /* gamma_z */
    { {0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0} },     /* gamma_t */
};
static const double GAMMA5[4] = { 1.0, 1.0, -1.0, -1.0 };           /* diagonal */
/* R2: P+- = (1 +- gamma5)/2, diagonal */
static const double PPLUS[4]  = { 1.0, 1.0, 0.0, 0.0 };
static const double PMINUS[4] = { 0.0, 0.0, 1.0, 1.0 };

void oracle_gamma(int mu, double* out_reim /* 4*4*2 */) {
    for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) {
        cplx g = (mu < 4) ? GAMMA[mu][a][b] : ((a == b) ? GAMMA5[a] : 0.0);
        out_reim[(a * 4 + b) * 2 + 0] = creal(g);
        out_reim[(a * 4 + b) * 2 + 1] = cimag(g);
    }
}

typedef struct {
    int L[4];       /* Lx, Ly, Lz, Lt */
    int Ls;
    int64_t V4;     /* 4D volume */
} geom_t;

static geom_t make_geom(const int* L, int Ls) {
    geom_t g;
    for (int i = 0; i < 4; i++) g.L[i] = L[i];
    g.Ls = Ls;
    g.V4 = (int64_t)L[0] * L[1] * L[2] * L[3];
    return g;
}

/* lexicographic 4D site index, x fastest (canonical order [t][z][y][x]) */
static inline int64_t site_index(const geom_t* g, const int c[4]) {
    return c[0] + (int64_t)g->L[0] * (c[1] + (int64_t)g->L[1] * (c[2] + (int64_t)g->L[2] * c[3]));
}
static inline void site_coords(const geom_t* g, int64_t idx, int c[4]) {
    for (int i = 0; i < 4; i++) { c[i] = (int)(idx % g->L[i]); idx /= g->L[i]; }
}
/* spinor element pointer: 12 complex at (rhs, s, site) */
static inline int64_t spinor_off(const geom_t* g, int rhs, int s, int64_t site) {
    return (((int64_t)rhs * g->Ls + s) * g->V4 + site) * 12;
}
static inline const cplx* link_ptr(const geom_t* g, const cplx* U, int mu, int64_t site) {
    return U + ((int64_t)mu * g->V4 + site) * 9;
}

/*
 * One non-zero block of D_hop (eq. 2) in row x:   block = sign * G (x) W
 *   forward  (dir=+1): column y = x+mu,  G = 1 - gamma_mu,  W = U_mu(x)
 *   backward (dir=-1): column y = x-mu,  G = 1 + gamma_mu,  W = U_mu^dag(y)
 * sign = -1 if the hop crosses the t seam (R3: antiperiodic in t, periodic in x,y,z), else +1.
 */
typedef struct { int64_t col; cplx G[4][4]; cplx W[3][3]; double sign; } hop_block_t;

static void hop_block(const geom_t* g, const cplx* U, int64_t x, int mu, int dir, hop_block_t* b) {
    int c[4], n[4];
    site_coords(g, x, c);
    for (int i = 0; i < 4; i++) n[i] = c[i];
    n[mu] = c[mu] + dir;
    b->sign = 1.0;
    if (n[mu] >= g->L[mu]) { n[mu] -= g->L[mu]; if (mu == 3) b->sign = -1.0; }
    if (n[mu] < 0)         { n[mu] += g->L[mu]; if (mu == 3) b->sign = -1.0; }
    b->col = site_index(g, n);
    for (int a = 0; a < 4; a++) for (int bb = 0; bb < 4; bb++)
        b->G[a][bb] = ((a == bb) ? 1.0 : 0.0) - (double)dir * GAMMA[mu][a][bb];
    if (dir > 0) {
        const cplx* u = link_ptr(g, U, mu, x);
        for (int a = 0; a < 3; a++) for (int bb = 0; bb < 3; bb++) b->W[a][bb] = u[a * 3 + bb];
    } else {
        const cplx* u = link_ptr(g, U, mu, b->col);
        for (int a = 0; a < 3; a++) for (int bb = 0; bb < 3; bb++) b->W[a][bb] = conj(u[bb * 3 + a]);
    }
}

/* out[12] += sign * (G (x) W) in[12]      (spin index outer, colour inner) */
static void block_apply(const hop_block_t* b, const cplx* in, cplx* out) {
    cplx tmp[4][3];
    for (int sp = 0; sp < 4; sp++) for (int a = 0; a < 3; a++) {
        cplx acc = 0;
        for (int c = 0; c < 3; c++) acc += b->W[a][c] * in[sp * 3 + c];
        tmp[sp][a] = acc;
    }
    for (int sp = 0; sp < 4; sp++) for (int a = 0; a < 3; a++) {
        cplx acc = 0;
        for (int sq = 0; sq < 4; sq++) acc += b->G[sp][sq] * tmp[sq][a];
        out[sp * 3 + a] += b->sign * acc;
    }
}
/* out[12] += sign * (G (x) W)^dagger in[12] */
static void block_apply_dag(const hop_block_t* b, const cplx* in, cplx* out) {
    cplx tmp[4][3];
    for (int sp = 0; sp < 4; sp++) for (int a = 0; a < 3; a++) {
        cplx acc = 0;
        for (int c = 0; c < 3; c++) acc += conj(b->W[c][a]) * in[sp * 3 + c];
        tmp[sp][a] = acc;
    }
    for (int sp = 0; sp < 4; sp++) for (int a = 0; a < 3; a++) {
        cplx acc = 0;
        for (int sq = 0; sq < 4; sq++) acc += conj(b->G[sq][sp]) * tmp[sq][a];
        out[sp * 3 + a] += b->sign * acc;
    }
}

/* ------------------------------------------------------------------------------------------
 * D_hop (eq. 2), optionally restricted to output rows of one 4D parity
 *   row_parity = -1 : all rows;  0/1 : only rows x with (x+y+z+t)%2 == row_parity (others: 0)
 *   dagger = 0 : out[x] = sum_blocks B(x,y) in[y]
 *   dagger = 1 : TRUE adjoint of the same (row-restricted) operator: out[y] += B(x,y)^dag in[x]
 * Acts independently on every s and rhs (D_hop is diagonal in the fifth dimension).
 * ------------------------------------------------------------------------------------------ */
static inline int parity_of(const geom_t* g, int64_t x) {
    int c[4]; site_coords(g, x, c); return (c[0] + c[1] + c[2] + c[3]) & 1;
}

static void dhop_core(const geom_t* g, const cplx* U, const cplx* in, cplx* out, int nrhs,
                      int row_parity, int dagger) {
    const int64_t nslice = (int64_t)nrhs * g->Ls;
    memset(out, 0, sizeof(cplx) * (size_t)(nslice * g->V4 * 12));
    if (!dagger) {
        #pragma omp parallel for collapse(2) schedule(static)
        for (int64_t sl = 0; sl < nslice; sl++) {
            for (int64_t x = 0; x < g->V4; x++) {
                if (row_parity >= 0 && parity_of(g, x) != row_parity) continue;
                const cplx* inS = in + sl * g->V4 * 12;
                cplx* o = out + (sl * g->V4 + x) * 12;
                for (int mu = 0; mu < 4; mu++) for (int dir = +1; dir >= -1; dir -= 2) {
                    hop_block_t b; hop_block(g, U, x, mu, dir, &b);
                    block_apply(&b, inS + b.col * 12, o);
                }
            }
        }
    } else {
        /* scatter: parallel over slices only (rows of one slice write into shared columns) */
        #pragma omp parallel for schedule(static)
        for (int64_t sl = 0; sl < nslice; sl++) {
            const cplx* inS = in + sl * g->V4 * 12;
            cplx* outS = out + sl * g->V4 * 12;
            for (int64_t x = 0; x < g->V4; x++) {
                if (row_parity >= 0 && parity_of(g, x) != row_parity) continue;
                for (int mu = 0; mu < 4; mu++) for (int dir = +1; dir >= -1; dir -= 2) {
                    hop_block_t b; hop_block(g, U, x, mu, dir, &b);
                    block_apply_dag(&b, inS + x * 12, outS + b.col * 12);
                }
            }
        }
    }
}

void oracle_dhop(const int* L, int Ls, const double* U, const double* in, double* out, int nrhs,
                 int row_parity, int dagger) {
    geom_t g = make_geom(L, Ls);
    dhop_core(&g, (const cplx*)U, (const cplx*)in, (cplx*)out, nrhs, row_parity, dagger);
}

/* ------------------------------------------------------------------------------------------
 * The fifth-dimension matrix of eq. 4 (L39) WITHOUT its D_par diagonal: blocks (row s, col s'):
 *   (s, s+1) = -P_-   for s <= Ls-2          (s, s-1) = -P_+   for s >= 1
 *   (0, Ls-1) = +m P_+                       (Ls-1, 0) = +m P_-
 * Returned as a list of (col, coefficient, projector diagonal) for a given row.
 * ------------------------------------------------------------------------------------------ */
typedef struct { int col; double coef; const double* P; } sblock_t;

static int s_row_blocks(int Ls, double mass, int s, sblock_t blk[4]) {
    int n = 0;
    if (s + 1 <= Ls - 1) { blk[n].col = s + 1; blk[n].coef = -1.0; blk[n].P = PMINUS; n++; }
    if (s - 1 >= 0)      { blk[n].col = s - 1; blk[n].coef = -1.0; blk[n].P = PPLUS;  n++; }
    if (s == 0)          { blk[n].col = Ls - 1; blk[n].coef = mass; blk[n].P = PPLUS;  n++; }
    if (s == Ls - 1)     { blk[n].col = 0;      blk[n].coef = mass; blk[n].P = PMINUS; n++; }
    return n;
}

/* out += (diag * 1 + S) in   restricted to sites of site_parity (-1: all); dagger: true adjoint.
 * S is site-diagonal in 4D, so the adjoint only transposes the s-matrix (P real diagonal). */
static void s_matrix_accum(const geom_t* g, double diag, double mass, const cplx* in, cplx* out,
                           int nrhs, int site_parity, int dagger) {
    #pragma omp parallel for collapse(2) schedule(static)
    for (int r = 0; r < nrhs; r++) {
        for (int64_t x = 0; x < g->V4; x++) {
            if (site_parity >= 0 && parity_of(g, x) != site_parity) continue;
            for (int s = 0; s < g->Ls; s++) {
                const cplx* i_row = in + spinor_off(g, r, s, x);
                cplx* o_row = out + spinor_off(g, r, s, x);
                for (int k = 0; k < 12; k++) o_row[k] += diag * i_row[k];
                sblock_t blk[4];
                int n = s_row_blocks(g->Ls, mass, s, blk);
                for (int j = 0; j < n; j++) {
                    if (!dagger) {      /* out[row s] += coef P in[col] */
                        const cplx* i_col = in + spinor_off(g, r, blk[j].col, x);
                        for (int sp = 0; sp < 4; sp++) for (int c = 0; c < 3; c++)
                            o_row[sp * 3 + c] += blk[j].coef * blk[j].P[sp] * i_col[sp * 3 + c];
                    } else {            /* out[col] += (coef P)^dag in[row s] */
                        cplx* o_col = out + spinor_off(g, r, blk[j].col, x);
                        for (int sp = 0; sp < 4; sp++) for (int c = 0; c < 3; c++)
                            o_col[sp * 3 + c] += blk[j].coef * blk[j].P[sp] * i_row[sp * 3 + c];
                    }
                }
            }
        }
    }
}

/* D_DW (eq. 4 L39 with eq. 5):  out = (5-M5) in - 1/2 D_hop in + S in ;  dagger: true adjoint */
static void ddw_core(const geom_t* g, double M5, double mass, const cplx* U, const cplx* in,
                     cplx* out, int nrhs, int dagger) {
    const int64_t n = (int64_t)nrhs * g->Ls * g->V4 * 12;
    dhop_core(g, U, in, out, nrhs, -1, dagger);
    for (int64_t i = 0; i < n; i++) out[i] *= -0.5;
    s_matrix_accum(g, 5.0 - M5, mass, in, out, nrhs, -1, dagger);
}

void oracle_ddw(const int* L, int Ls, double M5, double mass, const double* U, const double* in,
                double* out, int nrhs, int dagger) {
    geom_t g = make_geom(L, Ls);
    ddw_core(&g, M5, mass, (const cplx*)U, (const cplx*)in, (cplx*)out, nrhs, dagger);
}

/* D_W(M) = M + 4 - 1/2 D_hop (eq. 1); acts on each s slice independently. */
void oracle_dwilson(const int* L, int Ls, double M, const double* U, const double* in, double* out,
                    int nrhs) {
    geom_t g = make_geom(L, Ls);
    const int64_t n = (int64_t)nrhs * g.Ls * g.V4 * 12;
    cplx* o = (cplx*)out; const cplx* i_ = (const cplx*)in;
    dhop_core(&g, (const cplx*)U, i_, o, nrhs, -1, 0);
    for (int64_t i = 0; i < n; i++) o[i] = (M + 4.0) * i_[i] - 0.5 * o[i];
}

/* Gamma5 = gamma5 R5 (L46):  out(x,s) = gamma5 in(x, Ls-1-s)   (R6) */
static void gamma5r5_core(const geom_t* g, const cplx* in, cplx* out, int nrhs) {
    for (int r = 0; r < nrhs; r++) for (int s = 0; s < g->Ls; s++) for (int64_t x = 0; x < g->V4; x++) {
        const cplx* i_ = in + spinor_off(g, r, g->Ls - 1 - s, x);
        cplx* o = out + spinor_off(g, r, s, x);
        for (int sp = 0; sp < 4; sp++) for (int c = 0; c < 3; c++) o[sp * 3 + c] = GAMMA5[sp] * i_[sp * 3 + c];
    }
}
void oracle_gamma5r5(const int* L, int Ls, const double* in, double* out, int nrhs) {
    geom_t g = make_geom(L, Ls);
    gamma5r5_core(&g, (const cplx*)in, (cplx*)out, nrhs);
}

/* H_DW = Gamma5 D_DW (eq. 6) */
void oracle_hdw(const int* L, int Ls, double M5, double mass, const double* U, const double* in,
                double* out, int nrhs) {
    geom_t g = make_geom(L, Ls);
    const int64_t n = (int64_t)nrhs * g.Ls * g.V4 * 12;
    cplx* tmp = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    ddw_core(&g, M5, mass, (const cplx*)U, (const cplx*)in, tmp, nrhs, 0);
    gamma5r5_core(&g, tmp, (cplx*)out, nrhs);
    free(tmp);
}

/* D_PV = D_DW with unit mass parameter (L50, R7) */
void oracle_dpv(const int* L, int Ls, double M5, const double* U, const double* in, double* out,
                int nrhs, int dagger) {
    geom_t g = make_geom(L, Ls);
    ddw_core(&g, M5, 1.0, (const cplx*)U, (const cplx*)in, (cplx*)out, nrhs, dagger);
}

/* ------------------------------------------------------------------------------------------
 * Even-odd pieces (R8: 4D parity, even = 0; every s of a 4D site shares its parity).
 *   M_pp  = (5-M5) + S     restricted to sites of parity p        (site-diagonal in 4D)
 *   M_pq  = -1/2 D_hop     rows of parity p, columns parity q=1-p
 *   M_pc  = M_ee - M_eo M_oo^{-1} M_oe                            (Table V, R9)
 * ------------------------------------------------------------------------------------------ */

/* Dense Ls x Ls real matrix of M_pp for one spin component sp:  A[s][s'] (row-major). */
static void mpp_dense(int Ls, double M5, double mass, int sp, double* A) {
    for (int i = 0; i < Ls * Ls; i++) A[i] = 0.0;
    for (int s = 0; s < Ls; s++) {
        A[s * Ls + s] += 5.0 - M5;
        sblock_t blk[4];
        int n = s_row_blocks(Ls, mass, s, blk);
        for (int j = 0; j < n; j++) A[s * Ls + blk[j].col] += blk[j].coef * blk[j].P[sp];
    }
}

/* Generic dense inverse by Gauss-Jordan elimination with partial pivoting. Returns 0 on success. */
static int dense_inverse(int n, const double* A, double* Ainv) {
    double* w = (double*)malloc(sizeof(double) * (size_t)n * 2 * n);
    for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) {
        w[i * 2 * n + j] = A[i * n + j];
        w[i * 2 * n + n + j] = (i == j) ? 1.0 : 0.0;
    }
    for (int c = 0; c < n; c++) {
        int piv = c; double best = fabs(w[c * 2 * n + c]);
        for (int r = c + 1; r < n; r++) if (fabs(w[r * 2 * n + c]) > best) { best = fabs(w[r * 2 * n + c]); piv = r; }
        if (best == 0.0) { free(w); return -1; }
        if (piv != c) for (int j = 0; j < 2 * n; j++) { double t = w[c * 2 * n + j]; w[c * 2 * n + j] = w[piv * 2 * n + j]; w[piv * 2 * n + j] = t; }
        double inv = 1.0 / w[c * 2 * n + c];
        for (int j = 0; j < 2 * n; j++) w[c * 2 * n + j] *= inv;
        for (int r = 0; r < n; r++) if (r != c) {
            double f = w[r * 2 * n + c];
            if (f != 0.0) for (int j = 0; j < 2 * n; j++) w[r * 2 * n + j] -= f * w[c * 2 * n + j];
        }
    }
    for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) Ainv[i * n + j] = w[i * 2 * n + n + j];
    free(w);
    return 0;
}

/* out = M_pp^{-1} in on sites of site_parity (other sites: 0).  dagger: (M_pp^dag)^{-1}, i.e. the
 * inverse of the TRANSPOSED s-matrix (it is real).  Generic elimination, not a closed form. */
static int mpp_inv_core(const geom_t* g, double M5, double mass, const cplx* in, cplx* out, int nrhs,
                        int site_parity, int dagger) {
    const int Ls = g->Ls;
    double* A = (double*)malloc(sizeof(double) * (size_t)Ls * Ls);
    double* Ainv = (double*)malloc(sizeof(double) * (size_t)4 * Ls * Ls);
    for (int sp = 0; sp < 4; sp++) {
        mpp_dense(Ls, M5, mass, sp, A);
        if (dagger) for (int i = 0; i < Ls; i++) for (int j = i + 1; j < Ls; j++) { double t = A[i * Ls + j]; A[i * Ls + j] = A[j * Ls + i]; A[j * Ls + i] = t; }
        if (dense_inverse(Ls, A, Ainv + (size_t)sp * Ls * Ls)) { free(A); free(Ainv); return -1; }
    }
    memset(out, 0, sizeof(cplx) * (size_t)((int64_t)nrhs * Ls * g->V4 * 12));
    #pragma omp parallel for collapse(2) schedule(static)
    for (int r = 0; r < nrhs; r++) {
        for (int64_t x = 0; x < g->V4; x++) {
            if (site_parity >= 0 && parity_of(g, x) != site_parity) continue;
            for (int s = 0; s < Ls; s++) {
                cplx* o = out + spinor_off(g, r, s, x);
                for (int s2 = 0; s2 < Ls; s2++) {
                    const cplx* i_ = in + spinor_off(g, r, s2, x);
                    for (int sp = 0; sp < 4; sp++) {
                        double a = Ainv[((size_t)sp * Ls + s) * Ls + s2];
                        for (int c = 0; c < 3; c++) o[sp * 3 + c] += a * i_[sp * 3 + c];
                    }
                }
            }
        }
    }
    free(A); free(Ainv);
    return 0;
}

int oracle_mpp_inv(const int* L, int Ls, double M5, double mass, const double* in, double* out,
                   int nrhs, int site_parity, int dagger) {
    geom_t g = make_geom(L, Ls);
    return mpp_inv_core(&g, M5, mass, (const cplx*)in, (cplx*)out, nrhs, site_parity, dagger);
}

/* out = M_pp in  on sites of site_parity (other sites 0) */
void oracle_mpp(const int* L, int Ls, double M5, double mass, const double* in, double* out,
                int nrhs, int site_parity, int dagger) {
    geom_t g = make_geom(L, Ls);
    memset(out, 0, sizeof(cplx) * (size_t)((int64_t)nrhs * Ls * g.V4 * 12));
    s_matrix_accum(&g, 5.0 - M5, mass, (const cplx*)in, (cplx*)out, nrhs, site_parity, dagger);
}

/* M_pc psi_e = M_ee psi_e - M_eo M_oo^{-1} M_oe psi_e   (Table V), input/output: canonical
 * full arrays whose odd sites are zero / are written as zero.
 * dagger: M_pc^dag = M_ee^dag - M_oe^dag (M_oo^dag)^{-1} M_eo^dag, each factor a true adjoint.  */
static int mpc_core(const geom_t* g, double M5, double mass, const cplx* U, const cplx* in, cplx* out,
                    int nrhs, int dagger) {
    const int64_t n = (int64_t)nrhs * g->Ls * g->V4 * 12;
    cplx* t1 = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    cplx* t2 = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    int rc;
    if (!dagger) {
        dhop_core(g, U, in, t1, nrhs, /*rows odd*/1, 0);            /* t1 = D_hop_oe in  ; M_oe = -1/2 */
        for (int64_t i = 0; i < n; i++) t1[i] *= -0.5;
        rc = mpp_inv_core(g, M5, mass, t1, t2, nrhs, 1, 0);         /* t2 = M_oo^{-1} M_oe in */
        dhop_core(g, U, t2, t1, nrhs, /*rows even*/0, 0);           /* t1 = D_hop_eo t2 ; M_eo = -1/2 */
        for (int64_t i = 0; i < n; i++) t1[i] *= -0.5;
    } else {
        dhop_core(g, U, in, t1, nrhs, /*rows even*/0, 1);           /* t1 = (D_hop_eo)^dag in : even -> odd */
        for (int64_t i = 0; i < n; i++) t1[i] *= -0.5;
        rc = mpp_inv_core(g, M5, mass, t1, t2, nrhs, 1, 1);         /* (M_oo^dag)^{-1} */
        dhop_core(g, U, t2, t1, nrhs, /*rows odd*/1, 1);            /* (D_hop_oe)^dag : odd -> even */
        for (int64_t i = 0; i < n; i++) t1[i] *= -0.5;
    }
    memset(out, 0, sizeof(cplx) * (size_t)n);
    s_matrix_accum(g, 5.0 - M5, mass, in, out, nrhs, 0, dagger);    /* M_ee in (or its adjoint) */
    for (int64_t i = 0; i < n; i++) out[i] -= t1[i];
    free(t1); free(t2);
    return rc;
}

int oracle_mpc(const int* L, int Ls, double M5, double mass, const double* U, const double* in,
               double* out, int nrhs, int dagger) {
    geom_t g = make_geom(L, Ls);
    return mpc_core(&g, M5, mass, (const cplx*)U, (const cplx*)in, (cplx*)out, nrhs, dagger);
}

/* ---- BLAS-1 definitions (R18), per rhs ---- */
void oracle_inner(int64_t n_per_rhs, int nrhs, const double* x, const double* y, double* out /*2*nrhs*/) {
    const cplx* X = (const cplx*)x; const cplx* Y = (const cplx*)y;
    for (int r = 0; r < nrhs; r++) {
        cplx acc = 0;
        for (int64_t i = 0; i < n_per_rhs; i++) acc += conj(X[r * n_per_rhs + i]) * Y[r * n_per_rhs + i];
        out[2 * r] = creal(acc); out[2 * r + 1] = cimag(acc);
    }
}
void oracle_axpy(int64_t n_per_rhs, int nrhs, const double* a /*2*nrhs*/, const double* x, double* y) {
    const cplx* X = (const cplx*)x; cplx* Y = (cplx*)y;
    for (int r = 0; r < nrhs; r++) {
        cplx A = a[2 * r] + I * a[2 * r + 1];
        for (int64_t i = 0; i < n_per_rhs; i++) Y[r * n_per_rhs + i] += A * X[r * n_per_rhs + i];
    }
}

/* ------------------------------------------------------------------------------------------
 * Chebyshev filter (eq. 23; interval map L173; eq. 34 L227 with reading R10):
 *   X = 2 (A - lo) / (hi - lo) - 1,   A = M^dag M = D_DW^dag D_DW  (true adjoint; = H_DW^2 by eq. 11)
 *   t_0 = eta,  t_1 = X eta,  t_{k+1} = 2 X t_k - t_{k-1},   out = t_order            (R13, R14)
 * ------------------------------------------------------------------------------------------ */
static void apply_X(const geom_t* g, double M5, double mass, const cplx* U, double lo, double hi,
                    const cplx* in, cplx* out, cplx* tmp, int nrhs) {
    const int64_t n = (int64_t)nrhs * g->Ls * g->V4 * 12;
    ddw_core(g, M5, mass, U, in, tmp, nrhs, 0);
    ddw_core(g, M5, mass, U, tmp, out, nrhs, 1);
    for (int64_t i = 0; i < n; i++) out[i] = 2.0 * (out[i] - lo * in[i]) / (hi - lo) - in[i];
}

void oracle_chebyshev(const int* L, int Ls, double M5, double mass, const double* U, int order,
                      double lo, double hi, const double* in, double* out, int nrhs) {
    geom_t g = make_geom(L, Ls);
    const int64_t n = (int64_t)nrhs * g.Ls * g.V4 * 12;
    const cplx* eta = (const cplx*)in;
    cplx* tkm1 = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    cplx* tk   = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    cplx* xt   = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    cplx* tmp  = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    memcpy(tkm1, eta, sizeof(cplx) * (size_t)n);                       /* t_0 */
    if (order == 0) { memcpy(out, tkm1, sizeof(cplx) * (size_t)n); goto done; }
    apply_X(&g, M5, mass, (const cplx*)U, lo, hi, tkm1, tk, tmp, nrhs); /* t_1 */
    for (int k = 1; k < order; k++) {
        apply_X(&g, M5, mass, (const cplx*)U, lo, hi, tk, xt, tmp, nrhs);
        for (int64_t i = 0; i < n; i++) { cplx tnext = 2.0 * xt[i] - tkm1[i]; tkm1[i] = tk[i]; tk[i] = tnext; }
    }
    memcpy(out, tk, sizeof(cplx) * (size_t)n);
done:
    free(tkm1); free(tk); free(xt); free(tmp);
}

/* ------------------------------------------------------------------------------------------
 * Red-black CGNR (eq. 9): Hestenes-Stiefel CG [29] on A = M_pc^dag M_pc, fixed iteration
 * count, nrhs = 1.  b, x: canonical full arrays with odd sites zero.  x holds x_0 on entry.
 *   r_0 = b - A x_0, p_0 = r_0;  alpha = <r,r>/<p,Ap>; x += alpha p; r -= alpha Ap;
 *   beta = <r',r'>/<r,r>; p = r' + beta p.    hist[k] = |r_k|^2, k = 0..iters.
 * ------------------------------------------------------------------------------------------ */
static double norm2_all(const cplx* v, int64_t n) {
    double acc = 0; for (int64_t i = 0; i < n; i++) acc += creal(v[i]) * creal(v[i]) + cimag(v[i]) * cimag(v[i]);
    return acc;
}
static double re_inner_all(const cplx* a, const cplx* b, int64_t n) {
    double acc = 0; for (int64_t i = 0; i < n; i++) acc += creal(conj(a[i]) * b[i]);
    return acc;
}

int oracle_cg_schur(const int* L, int Ls, double M5, double mass, const double* U, const double* b_,
                    double* x_, int iters, double* hist) {
    geom_t g = make_geom(L, Ls);
    const int64_t n = (int64_t)g.Ls * g.V4 * 12;
    const cplx* b = (const cplx*)b_; cplx* x = (cplx*)x_; const cplx* Uc = (const cplx*)U;
    cplx* r = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    cplx* p = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    cplx* w = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    cplx* q = (cplx*)malloc(sizeof(cplx) * (size_t)n);
    int rc = mpc_core(&g, M5, mass, Uc, x, w, 1, 0);
    rc |= mpc_core(&g, M5, mass, Uc, w, q, 1, 1);
    for (int64_t i = 0; i < n; i++) { r[i] = b[i] - q[i]; p[i] = r[i]; }
    double rr = norm2_all(r, n);
    hist[0] = rr;
    for (int k = 0; k < iters; k++) {
        rc |= mpc_core(&g, M5, mass, Uc, p, w, 1, 0);      /* w = M p        */
        rc |= mpc_core(&g, M5, mass, Uc, w, q, 1, 1);      /* q = M^dag M p  */
        double pAp = re_inner_all(p, q, n);
        double alpha = rr / pAp;
        for (int64_t i = 0; i < n; i++) { x[i] += alpha * p[i]; r[i] -= alpha * q[i]; }
        double rr_new = norm2_all(r, n);
        double beta = rr_new / rr;
        for (int64_t i = 0; i < n; i++) p[i] = r[i] + beta * p[i];
        rr = rr_new;
        hist[k + 1] = rr;
    }
    free(r); free(p); free(w); free(q);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * Site-list mode: evaluate the DEFINITION of D_DW at a list of 4D sites only,
 * from gathered neighbourhoods, for lattices too big for a host-side full-volume oracle.
 *   coords[n][4]             (x,y,z,t) of each sampled output site
 *   nbr[n][9][Ls][12]        spinors: slot 0 = the site itself, slot 1+2*mu = x+mu, 2+2*mu = x-mu
 *   links[n][8][9]           slot 2*mu = U_mu(x), slot 2*mu+1 = U_mu(x-mu)   (as stored, undaggered)
 *   out[n][Ls][12]
 * ------------------------------------------------------------------------------------------ */
void oracle_ddw_sites(const int* L, int Ls, double M5, double mass, int64_t n, const int* coords,
                      const double* nbr_, const double* links_, double* out_) {
    const cplx* nbr = (const cplx*)nbr_; const cplx* links = (const cplx*)links_; cplx* out = (cplx*)out_;
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; i++) {
        const int* c = coords + 4 * i;
        for (int s = 0; s < Ls; s++) {
            cplx hop[12]; for (int k = 0; k < 12; k++) hop[k] = 0;
            for (int mu = 0; mu < 4; mu++) for (int dir = +1; dir >= -1; dir -= 2) {
                hop_block_t b; b.col = 0; b.sign = 1.0;
                int nc = c[mu] + dir;
                if ((nc >= L[mu] || nc < 0) && mu == 3) b.sign = -1.0;
                for (int a = 0; a < 4; a++) for (int bb = 0; bb < 4; bb++)
                    b.G[a][bb] = ((a == bb) ? 1.0 : 0.0) - (double)dir * GAMMA[mu][a][bb];
                const cplx* u = links + (i * 8 + 2 * mu + (dir > 0 ? 0 : 1)) * 9;
                for (int a = 0; a < 3; a++) for (int bb = 0; bb < 3; bb++)
                    b.W[a][bb] = (dir > 0) ? u[a * 3 + bb] : conj(u[bb * 3 + a]);
                const cplx* src = nbr + ((i * 9 + 1 + 2 * mu + (dir > 0 ? 0 : 1)) * Ls + s) * 12;
                block_apply(&b, src, hop);
            }
            const cplx* self = nbr + ((i * 9 + 0) * Ls) * 12;
            cplx* o = out + (i * Ls + s) * 12;
            for (int k = 0; k < 12; k++) o[k] = (5.0 - M5) * self[s * 12 + k] - 0.5 * hop[k];
            sblock_t blk[4];
            int nb = s_row_blocks(Ls, mass, s, blk);
            for (int j = 0; j < nb; j++) for (int sp = 0; sp < 4; sp++) for (int cc = 0; cc < 3; cc++)
                o[sp * 3 + cc] += blk[j].coef * blk[j].P[sp] * self[blk[j].col * 12 + sp * 3 + cc];
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Site-list mode for the Schur operator (Table V): evaluate
 *   M_pc psi_e = M_ee psi_e - M_eo M_oo^{-1} M_oe psi_e      (M_eo = M_oe = -1/2 D_hop, R8/R9)
 * at a list of EVEN 4D sites x from gathered neighbourhoods: the 8 odd neighbours y_d of x and,
 * for each of them, its 8 even neighbours z_{d,e} (the 33 even sites at taxicab distance 0 or 2,
 * passed with repetition so that the loops below stay the plain definition).
 * Direction slots: d, e = 2*mu (+mu) or 2*mu+1 (-mu).
 *   coords[n][4]           (x,y,z,t) of x
 *   self[n][Ls][12]        psi_e(x)
 *   nbr2[n][8][8][Ls][12]  psi_e(z_{d,e}),  y_d = x + d,  z_{d,e} = y_d + e
 *   links1[n][8][9]        slot 2*mu = U_mu(x),   2*mu+1 = U_mu(x - mu)        (as stored, undaggered)
 *   links2[n][8][8][9]     [d] slot 2*nu = U_nu(y_d), 2*nu+1 = U_nu(y_d - nu)
 *   out[n][Ls][12]
 * M_oo^{-1}: generic elimination of the dense Ls x Ls s-matrix (dense_inverse), as in mpp_inv_core.
 * dagger: M_pc^dag = M_ee^dag - M_oe^dag (M_oo^dag)^{-1} M_eo^dag with every factor a true adjoint:
 * the block B(row, col) of the FORWARD operator is built from its definition and applied as B^dag
 * from row to col (block_apply_dag), exactly as dhop_core does on full arrays.
 * ------------------------------------------------------------------------------------------ */
static void sites_block(const int* L, const int c_row[4], int mu, int dir, const cplx* u_fwd /* U_mu(row) */,
                        const cplx* u_bwd /* U_mu(row - mu) */, hop_block_t* b) {
    b->col = 0; b->sign = 1.0;
    const int nc = c_row[mu] + dir;
    if ((nc >= L[mu] || nc < 0) && mu == 3) b->sign = -1.0;
    for (int a = 0; a < 4; a++) for (int bb = 0; bb < 4; bb++)
        b->G[a][bb] = ((a == bb) ? 1.0 : 0.0) - (double)dir * GAMMA[mu][a][bb];
    for (int a = 0; a < 3; a++) for (int bb = 0; bb < 3; bb++)
        b->W[a][bb] = (dir > 0) ? u_fwd[a * 3 + bb] : conj(u_bwd[bb * 3 + a]);
}

int oracle_mpc_sites(const int* L, int Ls, double M5, double mass, int64_t n, const int* coords,
                     const double* self_, const double* nbr2_, const double* links1_, const double* links2_,
                     double* out_, int dagger) {
    const cplx* self = (const cplx*)self_; const cplx* nbr2 = (const cplx*)nbr2_;
    const cplx* links1 = (const cplx*)links1_; const cplx* links2 = (const cplx*)links2_; cplx* out = (cplx*)out_;
    double* A = (double*)malloc(sizeof(double) * (size_t)Ls * Ls);
    double* Ainv = (double*)malloc(sizeof(double) * (size_t)4 * Ls * Ls);
    for (int sp = 0; sp < 4; sp++) {
        mpp_dense(Ls, M5, mass, sp, A);
        if (dagger) for (int i = 0; i < Ls; i++) for (int j = i + 1; j < Ls; j++) { double t = A[i * Ls + j]; A[i * Ls + j] = A[j * Ls + i]; A[j * Ls + i] = t; }
        if (dense_inverse(Ls, A, Ainv + (size_t)sp * Ls * Ls)) { free(A); free(Ainv); return -1; }
    }
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; i++) {
        const int* cx = coords + 4 * i;
        cplx* acc = (cplx*)calloc((size_t)Ls * 12, sizeof(cplx));      /* D_hop-type sum over the odd neighbours, row x */
        cplx* ty = (cplx*)malloc(sizeof(cplx) * (size_t)Ls * 12);
        cplx* vy = (cplx*)malloc(sizeof(cplx) * (size_t)Ls * 12);
        for (int d = 0; d < 8; d++) {
            const int mu = d / 2, dir = (d % 2 == 0) ? +1 : -1;
            int cy[4] = {cx[0], cx[1], cx[2], cx[3]};
            cy[mu] = (cx[mu] + dir + L[mu]) % L[mu];
            /* ty = M_oe psi (or M_eo^dag psi) at the odd site y_d */
            for (int k = 0; k < Ls * 12; k++) ty[k] = 0;
            for (int e = 0; e < 8; e++) {
                const int nu = e / 2, dire = (e % 2 == 0) ? +1 : -1;
                const cplx* l2 = links2 + ((i * 8 + d) * 8) * 9;
                const cplx* uy = l2 + (2 * nu) * 9;                 /* U_nu(y)      */
                const cplx* uym = l2 + (2 * nu + 1) * 9;            /* U_nu(y - nu) */
                const cplx* psi_z = nbr2 + (((i * 8 + d) * 8 + e) * (int64_t)Ls) * 12;
                hop_block_t b;
                if (!dagger) {
                    sites_block(L, cy, nu, dire, uy, uym, &b);      /* B(row y, col z = y + e) */
                    for (int s = 0; s < Ls; s++) block_apply(&b, psi_z + s * 12, ty + s * 12);
                } else {
                    /* B(row z, col y) of the forward operator: from z the site y lies in direction (nu, -dire);
                     * U_nu(z) = U_nu(y - nu) when z = y - nu, U_nu(z - nu) = U_nu(y) when z = y + nu */
                    int cz[4] = {cy[0], cy[1], cy[2], cy[3]};
                    cz[nu] = (cy[nu] + dire + L[nu]) % L[nu];
                    sites_block(L, cz, nu, -dire, uym, uy, &b);
                    for (int s = 0; s < Ls; s++) block_apply_dag(&b, psi_z + s * 12, ty + s * 12);
                }
            }
            for (int k = 0; k < Ls * 12; k++) ty[k] *= -0.5;
            /* vy = M_oo^{-1} ty  (or (M_oo^dag)^{-1}) */
            for (int s = 0; s < Ls; s++) for (int sp = 0; sp < 4; sp++) for (int c = 0; c < 3; c++) {
                cplx a = 0;
                for (int s2 = 0; s2 < Ls; s2++) a += Ainv[((size_t)sp * Ls + s) * Ls + s2] * ty[s2 * 12 + sp * 3 + c];
                vy[s * 12 + sp * 3 + c] = a;
            }
            /* row x of D_hop_eo (or of D_hop_oe^dag) applied to vy */
            const cplx* ux = links1 + (i * 8 + 2 * mu) * 9;         /* U_mu(x)      */
            const cplx* uxm = links1 + (i * 8 + 2 * mu + 1) * 9;    /* U_mu(x - mu) */
            hop_block_t b;
            if (!dagger) {
                sites_block(L, cx, mu, dir, ux, uxm, &b);           /* B(row x, col y_d) */
                for (int s = 0; s < Ls; s++) block_apply(&b, vy + s * 12, acc + s * 12);
            } else {
                sites_block(L, cy, mu, -dir, uxm, ux, &b);          /* B(row y_d, col x): U_mu(y) = U_mu(x - mu) when y = x - mu, U_mu(y - mu) = U_mu(x) when y = x + mu */
                for (int s = 0; s < Ls; s++) block_apply_dag(&b, vy + s * 12, acc + s * 12);
            }
        }
        /* out = M_ee psi(x) - (-1/2) acc ;  M_ee = (5 - M5) + S  (adjoint: S transposed, scatter form) */
        const cplx* sx = self + (i * (int64_t)Ls) * 12;
        cplx* o = out + (i * (int64_t)Ls) * 12;
        for (int k = 0; k < Ls * 12; k++) o[k] = (5.0 - M5) * sx[k] + 0.5 * acc[k];
        for (int s = 0; s < Ls; s++) {
            sblock_t blk[4];
            const int nb = s_row_blocks(Ls, mass, s, blk);
            for (int j = 0; j < nb; j++) for (int sp = 0; sp < 4; sp++) for (int c = 0; c < 3; c++) {
                if (!dagger) o[s * 12 + sp * 3 + c] += blk[j].coef * blk[j].P[sp] * sx[blk[j].col * 12 + sp * 3 + c];
                else         o[blk[j].col * 12 + sp * 3 + c] += blk[j].coef * blk[j].P[sp] * sx[s * 12 + sp * 3 + c];
            }
        }
        free(acc); free(ty); free(vy);
    }
    free(A); free(Ainv);
    return 0;
}
