/*
 * rgf_oracle.c -- CPU ORACLE for the recursive Green's function (RGF) sweep.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or helper with the CUDA path
 * (paper_1107_5300_b200/csrc) and neither includes the other.
 *
 * What it computes (plain double precision, complex128, naive O(n^3) loops, its own
 * pivoted LU, no BLAS/LAPACK):
 *
 *   T(E) = Re Tr[ Gamma_L  G^dagger  Gamma_R  G ],   G = block (L-1, 0) of
 *          ( z - H_device - Sigma_L (+) 0 (+) Sigma_R )^-1 ,  z = E + i*eta
 *
 *   PAPER.md:33-37  Eq. 1  G = (E - H)^-1
 *   PAPER.md:37-41  Eq. 2  conductance = (2e^2/h) Tr[Gamma_L G^a Gamma_R G^r]
 *   PAPER.md:41-53  Eq. 3-5 slice recursion (Dyson equation), "G_1M ~ G^r"
 *   PAPER.md:53,58  lead self-energies at the first and last slice
 *   BASELINE.json:north_star  direct form G_ii = (z - H_i - V G_{i-1,i-1} V)^-1,
 *                             G_{i,1} = G_ii V G_{i-1,1}; Sancho-Rubio on the 2-slice cell
 *
 * Conventions (readings listed in DESIGN.md):
 *   device slices i = 0..L-1, atoms j = 0..M-1 (M = atoms per slice, L = #slices);
 *   H_i = diag(onsite[i][:]) + t on the sub/super diagonal (bond j<->j+1 removed if either
 *   end is a vacancy);  V_{i,i+1} = t*diag(m_i), m_i[j] = 1 iff (i+j) even, removed when the
 *   atom at either end is a vacancy; leads are clean (zero on-site, no vacancies) and
 *   continue the same parity rule: left lead = slices -1,-2,..., right lead = L,L+1,...
 *
 * Complex arrays cross this ABI as interleaved (re,im) doubles, row-major.
 *
 * orc_ldos_batch (O9) adds the diagonal blocks of the connected G (local density of states).
 *
 * parity pins (tests/test_oracle_pins.py): closed-form subband transmission of the clean
 * ribbon, brute-force inversion of the whole device (orc_transmission_brute), reciprocity
 * (orc_transmission with direction=1), bipartite / gauge symmetries, lead fixed-point
 * residual, LU against LAPACK, block-form lead == cell-form lead.
 * Disordered large configs have no value fixed by the paper: "parity unpinned" for those
 * (held by the invariants above only) -- see DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { double re, im; } cplx;

static inline cplx c_make(double re, double im) { cplx r; r.re = re; r.im = im; return r; }
static inline cplx c_add(cplx a, cplx b) { return c_make(a.re + b.re, a.im + b.im); }
static inline cplx c_sub(cplx a, cplx b) { return c_make(a.re - b.re, a.im - b.im); }
static inline cplx c_mul(cplx a, cplx b) { return c_make(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
static inline cplx c_scale(cplx a, double s) { return c_make(a.re * s, a.im * s); }
static inline double c_abs2(cplx a) { return a.re * a.re + a.im * a.im; }
/* a / b, Smith's algorithm (no overflow for the magnitudes met here, plain enough to read) */
static inline cplx c_div(cplx a, cplx b)
{
    if (fabs(b.re) >= fabs(b.im)) {
        double r = b.im / b.re, d = b.re + b.im * r;
        return c_make((a.re + a.im * r) / d, (a.im - a.re * r) / d);
    } else {
        double r = b.re / b.im, d = b.re * r + b.im;
        return c_make((a.re * r + a.im) / d, (a.im * r - a.re) / d);
    }
}

enum { ORC_OK = 0, ORC_EINVAL = -1, ORC_ENOMEM = -3, ORC_ENOCONV = -4, ORC_ESINGULAR = -5 };

/* ------------------------------------------------------------------------------------------
 * Dense helpers: naive matmul and naive LU inverse.
 * ---------------------------------------------------------------------------------------- */

/* C = A * B, all n x n, plain triple loop (i, k, j order so the inner loop is contiguous). */
static void mat_mul(int n, const cplx *A, const cplx *B, cplx *C)
{
    for (int i = 0; i < n; i++) {
        cplx *Ci = C + (size_t)i * n;
        for (int j = 0; j < n; j++) Ci[j] = c_make(0.0, 0.0);
        for (int k = 0; k < n; k++) {
            cplx a = A[(size_t)i * n + k];
            const cplx *Bk = B + (size_t)k * n;
            for (int j = 0; j < n; j++) Ci[j] = c_add(Ci[j], c_mul(a, Bk[j]));
        }
    }
}

/* Ainv = A^-1 by LU with partial (row) pivoting, then one forward/backward solve per unit
 * vector.  A is not modified.  Returns ORC_ESINGULAR on a zero / non-finite pivot.
 * ("one call of the linear equation solver" per recursion loop.) */
static int mat_inverse(int n, const cplx *A, cplx *Ainv)
{
    cplx *LU = (cplx *)malloc(sizeof(cplx) * (size_t)n * n);
    int *perm = (int *)malloc(sizeof(int) * (size_t)n);
    cplx *y = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    if (!LU || !perm || !y) { free(LU); free(perm); free(y); return ORC_ENOMEM; }
    memcpy(LU, A, sizeof(cplx) * (size_t)n * n);
    for (int i = 0; i < n; i++) perm[i] = i;
    int rc = ORC_OK;
    for (int k = 0; k < n; k++) {
        int p = k;
        double best = c_abs2(LU[(size_t)k * n + k]);
        for (int i = k + 1; i < n; i++) {
            double v = c_abs2(LU[(size_t)i * n + k]);
            if (v > best) { best = v; p = i; }
        }
        if (!(best > 0.0) || !isfinite(best)) { rc = ORC_ESINGULAR; break; }
        if (p != k) {
            for (int j = 0; j < n; j++) {
                cplx tmp = LU[(size_t)k * n + j];
                LU[(size_t)k * n + j] = LU[(size_t)p * n + j];
                LU[(size_t)p * n + j] = tmp;
            }
            int tp = perm[k]; perm[k] = perm[p]; perm[p] = tp;
        }
        cplx piv = LU[(size_t)k * n + k];
        for (int i = k + 1; i < n; i++) {
            cplx f = c_div(LU[(size_t)i * n + k], piv);
            LU[(size_t)i * n + k] = f;
            cplx *Li = LU + (size_t)i * n;
            const cplx *Lk = LU + (size_t)k * n;
            for (int j = k + 1; j < n; j++) Li[j] = c_sub(Li[j], c_mul(f, Lk[j]));
        }
    }
    if (rc == ORC_OK) {
        /* P A = L U.  Column c of A^-1 solves A x = e_c  <=>  L U x = P e_c. */
        for (int c = 0; c < n; c++) {
            for (int i = 0; i < n; i++) {
                cplx s = (perm[i] == c) ? c_make(1.0, 0.0) : c_make(0.0, 0.0);
                const cplx *Li = LU + (size_t)i * n;
                for (int j = 0; j < i; j++) s = c_sub(s, c_mul(Li[j], y[j]));
                y[i] = s;
            }
            for (int i = n - 1; i >= 0; i--) {
                cplx s = y[i];
                const cplx *Ui = LU + (size_t)i * n;
                for (int j = i + 1; j < n; j++) s = c_sub(s, c_mul(Ui[j], y[j]));
                y[i] = c_div(s, Ui[i]);
            }
            for (int i = 0; i < n; i++) Ainv[(size_t)i * n + c] = y[i];
        }
    }
    free(LU); free(perm); free(y);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O1. Operators of the armchair ribbon (BASELINE.json:configs[0]).
 * ---------------------------------------------------------------------------------------- */

/* m_i[j] = 1 iff (i + j) even; bit test so that negative (lead) slice indices work. */
static inline int mask_bit(int i, int j) { return (((i + j) & 1) == 0) ? 1 : 0; }

static inline int is_vacant(const uint8_t *vac, int M, int L, int i, int j)
{
    if (!vac || i < 0 || i >= L) return 0;        /* leads have no vacancies */
    return vac[(size_t)i * M + j] ? 1 : 0;
}

/* Inter-slice bond mask between slices i and i+1 (either may be a lead slice):
 * m'_i[j] = m_i[j] * !vac[i][j] * !vac[i+1][j]. */
static void bond_mask(int M, int L, const uint8_t *vac, int i, double *mprime)
{
    for (int j = 0; j < M; j++)
        mprime[j] = (mask_bit(i, j) && !is_vacant(vac, M, L, i, j) && !is_vacant(vac, M, L, i + 1, j)) ? 1.0 : 0.0;
}

/* Dense slice Hamiltonian H_i (M x M, real symmetric, stored complex).  onsite_i == NULL
 * gives the clean lead slice (zero on-site, all bonds). */
static void slice_hamiltonian(int M, int L, const double *onsite, const uint8_t *vac, int i, double t, cplx *H)
{
    for (size_t k = 0; k < (size_t)M * M; k++) H[k] = c_make(0.0, 0.0);
    int in_device = (i >= 0 && i < L && onsite != NULL);
    for (int j = 0; j < M; j++) {
        H[(size_t)j * M + j] = c_make(in_device ? onsite[(size_t)i * M + j] : 0.0, 0.0);
        if (j + 1 < M && !is_vacant(vac, M, L, i, j) && !is_vacant(vac, M, L, i, j + 1)) {
            H[(size_t)j * M + j + 1] = c_make(t, 0.0);
            H[(size_t)(j + 1) * M + j] = c_make(t, 0.0);
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * O2/O3. Lead surface Green's function by Sancho-Rubio decimation
 * (BASELINE.json:north_star "Sancho-Rubio decimation on the clean two-slice lead cell";
 *  PAPER.md:53 "at the 1-st and M-th slices, one should also find and include the
 *  self-energies due to the leads").
 *
 * Cell form (the definition used for pins): the lead is a chain of identical 2-slice
 * cells; h00 = [[H_c, V_a],[V_a, H_c]] (2M x 2M), h01 = [[0,0],[V_b,0]] couples the second
 * slice of cell n to the first slice of cell n+1.  alpha = h01, beta = h01^T,
 * eps = eps_s = h00; repeat { g = (z-eps)^-1; eps_s += (towards the bulk) ;
 * eps += alpha g beta + beta g alpha; alpha <- alpha g alpha; beta <- beta g beta }
 * until max|alpha|, max|beta| < tol.  For the right lead the bulk lies at +n, so
 * eps_s += alpha g beta and the surface slice is the FIRST slice of the cell (top-left
 * block); for the left lead the bulk lies at -n, eps_s += beta g alpha and the surface
 * slice is the SECOND slice (bottom-right block).
 * ---------------------------------------------------------------------------------------- */
#define ORC_SR_TOL 1e-14
#define ORC_SR_MAXIT 64

static double max_abs(size_t n, const cplx *A)
{
    double m = 0.0;
    for (size_t k = 0; k < n; k++) { double v = sqrt(c_abs2(A[k])); if (v > m) m = v; }
    return m;
}

/* va[j], vb[j]: diagonals of V_a (inside the cell) and V_b (between cells), already times t.
 * side = +1 right lead, -1 left lead.  g_out = M x M surface block. */
static int lead_surface_cell(int M, double t, cplx z, const double *va, const double *vb, int side, cplx *g_out, int *iters_out)
{
    int N = 2 * M;
    size_t NN = (size_t)N * N;
    cplx *buf = (cplx *)malloc(sizeof(cplx) * NN * 9);
    if (!buf) return ORC_ENOMEM;
    cplx *eps = buf, *eps_s = buf + NN, *alpha = buf + 2 * NN, *beta = buf + 3 * NN, *g = buf + 4 * NN;
    cplx *T1 = buf + 5 * NN, *T2 = buf + 6 * NN, *T3 = buf + 7 * NN, *W = buf + 8 * NN;
    cplx *Hc = (cplx *)malloc(sizeof(cplx) * (size_t)M * M);
    if (!Hc) { free(buf); return ORC_ENOMEM; }
    slice_hamiltonian(M, 0, NULL, NULL, 0, t, Hc);
    for (size_t k = 0; k < NN; k++) { eps[k] = c_make(0, 0); alpha[k] = c_make(0, 0); beta[k] = c_make(0, 0); }
    for (int r = 0; r < M; r++)
        for (int c = 0; c < M; c++) {
            eps[(size_t)r * N + c] = Hc[(size_t)r * M + c];
            eps[(size_t)(M + r) * N + (M + c)] = Hc[(size_t)r * M + c];
        }
    for (int j = 0; j < M; j++) {
        eps[(size_t)j * N + (M + j)] = c_make(va[j], 0.0);
        eps[(size_t)(M + j) * N + j] = c_make(va[j], 0.0);
        alpha[(size_t)(M + j) * N + j] = c_make(vb[j], 0.0);   /* h01: second slice -> next cell's first */
        beta[(size_t)j * N + (M + j)] = c_make(vb[j], 0.0);    /* h01^T */
    }
    memcpy(eps_s, eps, sizeof(cplx) * NN);
    int rc = ORC_ENOCONV, it = 0;
    for (it = 0; it < ORC_SR_MAXIT; it++) {
        if (max_abs(NN, alpha) < ORC_SR_TOL && max_abs(NN, beta) < ORC_SR_TOL) { rc = ORC_OK; break; }
        for (size_t k = 0; k < NN; k++) W[k] = c_make(-eps[k].re, -eps[k].im);
        for (int d = 0; d < N; d++) W[(size_t)d * N + d] = c_add(W[(size_t)d * N + d], z);
        int r2 = mat_inverse(N, W, g);
        if (r2 != ORC_OK) { rc = r2; break; }
        mat_mul(N, alpha, g, T1);          /* alpha g */
        mat_mul(N, T1, beta, T2);          /* alpha g beta */
        mat_mul(N, beta, g, T3);           /* beta g */
        mat_mul(N, T3, alpha, W);          /* beta g alpha */
        for (size_t k = 0; k < NN; k++) {
            eps[k] = c_add(eps[k], c_add(T2[k], W[k]));
            eps_s[k] = c_add(eps_s[k], side > 0 ? T2[k] : W[k]);
        }
        mat_mul(N, T1, alpha, T2);         /* alpha g alpha */
        mat_mul(N, T3, beta, W);           /* beta g beta */
        memcpy(alpha, T2, sizeof(cplx) * NN);
        memcpy(beta, W, sizeof(cplx) * NN);
    }
    if (rc == ORC_OK) {
        for (size_t k = 0; k < NN; k++) W[k] = c_make(-eps_s[k].re, -eps_s[k].im);
        for (int d = 0; d < N; d++) W[(size_t)d * N + d] = c_add(W[(size_t)d * N + d], z);
        rc = mat_inverse(N, W, g);
        if (rc == ORC_OK) {
            int off = side > 0 ? 0 : M;
            for (int r = 0; r < M; r++)
                for (int c = 0; c < M; c++) g_out[(size_t)r * M + c] = g[(size_t)(off + r) * N + (off + c)];
        }
    }
    if (iters_out) *iters_out = it;
    free(buf); free(Hc);
    return rc;
}

/* Block form: the same semi-infinite chain with the non-surface slice of every cell
 * eliminated exactly first (G1 = (z - H_c)^-1), leaving a chain of M x M sites
 *   eps_s = H_c + V_a G1 V_a,  eps = eps_s + V_b G1 V_b,  alpha = V_a G1 V_b, beta = alpha^T
 * to which the same decimation is applied; the surface slice couples to the bulk through V_a
 * first for both leads, so side does not enter.  8x fewer flops than the cell form; pinned
 * against it in tests/test_oracle_pins.py. */
static int lead_surface_block(int M, double t, cplx z, const double *va, const double *vb, cplx *g_out, int *iters_out)
{
    size_t MM = (size_t)M * M;
    cplx *buf = (cplx *)malloc(sizeof(cplx) * MM * 10);
    if (!buf) return ORC_ENOMEM;
    cplx *eps = buf, *eps_s = buf + MM, *alpha = buf + 2 * MM, *beta = buf + 3 * MM, *g = buf + 4 * MM;
    cplx *T1 = buf + 5 * MM, *T2 = buf + 6 * MM, *T3 = buf + 7 * MM, *W = buf + 8 * MM, *Hc = buf + 9 * MM;
    slice_hamiltonian(M, 0, NULL, NULL, 0, t, Hc);
    for (size_t k = 0; k < MM; k++) W[k] = c_make(-Hc[k].re, -Hc[k].im);
    for (int d = 0; d < M; d++) W[(size_t)d * M + d] = c_add(W[(size_t)d * M + d], z);
    int rc = mat_inverse(M, W, g);           /* G1 */
    if (rc != ORC_OK) { free(buf); return rc; }
    for (int r = 0; r < M; r++)
        for (int c = 0; c < M; c++) {
            cplx G1 = g[(size_t)r * M + c];
            eps_s[(size_t)r * M + c] = c_add(Hc[(size_t)r * M + c], c_scale(G1, va[r] * va[c]));
            eps[(size_t)r * M + c] = c_add(eps_s[(size_t)r * M + c], c_scale(G1, vb[r] * vb[c]));
            alpha[(size_t)r * M + c] = c_scale(G1, va[r] * vb[c]);
        }
    for (int r = 0; r < M; r++)
        for (int c = 0; c < M; c++) beta[(size_t)r * M + c] = alpha[(size_t)c * M + r];
    rc = ORC_ENOCONV;
    int it;
    for (it = 0; it < ORC_SR_MAXIT; it++) {
        if (max_abs(MM, alpha) < ORC_SR_TOL && max_abs(MM, beta) < ORC_SR_TOL) { rc = ORC_OK; break; }
        for (size_t k = 0; k < MM; k++) W[k] = c_make(-eps[k].re, -eps[k].im);
        for (int d = 0; d < M; d++) W[(size_t)d * M + d] = c_add(W[(size_t)d * M + d], z);
        int r2 = mat_inverse(M, W, g);
        if (r2 != ORC_OK) { rc = r2; break; }
        mat_mul(M, alpha, g, T1);
        mat_mul(M, T1, beta, T2);          /* alpha g beta */
        mat_mul(M, beta, g, T3);
        mat_mul(M, T3, alpha, W);          /* beta g alpha */
        for (size_t k = 0; k < MM; k++) {
            eps[k] = c_add(eps[k], c_add(T2[k], W[k]));
            eps_s[k] = c_add(eps_s[k], T2[k]);
        }
        mat_mul(M, T1, alpha, T2);
        mat_mul(M, T3, beta, W);
        memcpy(alpha, T2, sizeof(cplx) * MM);
        memcpy(beta, W, sizeof(cplx) * MM);
    }
    if (rc == ORC_OK) {
        for (size_t k = 0; k < MM; k++) W[k] = c_make(-eps_s[k].re, -eps_s[k].im);
        for (int d = 0; d < M; d++) W[(size_t)d * M + d] = c_add(W[(size_t)d * M + d], z);
        rc = mat_inverse(M, W, g_out);
    }
    if (iters_out) *iters_out = it;
    free(buf);
    return rc;
}

/* Surface Green's function of one lead.  side=+1: right lead, surface slice = L, cell =
 * (L, L+1): V_a = t diag(m_L), V_b = t diag(m_{L+1}).  side=-1: left lead, surface slice =
 * -1, cell = (-2,-1): V_a = t diag(m_{-2}), V_b = t diag(m_{-1}) (coupling -1 -> 0, which
 * by periodicity equals -3 -> -2).  method 0 = cell form (2M x 2M), 1 = block form. */
static int lead_surface(int M, int L, double t, cplx z, int side, int method, cplx *g_out, int *iters_out)
{
    double *va = (double *)malloc(sizeof(double) * 2 * (size_t)M);
    if (!va) return ORC_ENOMEM;
    double *vb = va + M;
    for (int j = 0; j < M; j++) {
        if (side > 0) { va[j] = t * mask_bit(L, j); vb[j] = t * mask_bit(L + 1, j); }
        else          { va[j] = t * mask_bit(-2, j); vb[j] = t * mask_bit(-1, j); }
    }
    int rc = (method == 0) ? lead_surface_cell(M, t, z, va, vb, side, g_out, iters_out)
                           : lead_surface_block(M, t, z, va, vb, g_out, iters_out);
    free(va);
    return rc;
}

/* Sigma = V g_surf V with V = t diag(m') the (vacancy-aware) bond mask between the lead's
 * surface slice and the device's end slice (O2/O3). */
static int lead_self_energy(int M, int L, const uint8_t *vac, double t, cplx z, int side, int method, cplx *Sigma, int *iters_out)
{
    size_t MM = (size_t)M * M;
    cplx *g = (cplx *)malloc(sizeof(cplx) * MM);
    double *mp = (double *)malloc(sizeof(double) * (size_t)M);
    if (!g || !mp) { free(g); free(mp); return ORC_ENOMEM; }
    int rc = lead_surface(M, L, t, z, side, method, g, iters_out);
    if (rc == ORC_OK) {
        bond_mask(M, L, vac, side > 0 ? L - 1 : -1, mp);
        for (int r = 0; r < M; r++)
            for (int c = 0; c < M; c++)
                Sigma[(size_t)r * M + c] = c_scale(g[(size_t)r * M + c], (t * mp[r]) * (t * mp[c]));
    }
    free(g); free(mp);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O4-O6. The sweep and the trace.
 * direction 0: start at slice 0, end at L-1, propagate G_{i,0} (north_star's column form;
 *              the paper's Eq. 5 propagates the row G_{1j}, its transpose -- reading Q4).
 * direction 1: mirror sweep from slice L-1 down to 0 with the roles of the leads swapped,
 *              propagating G_{i,L-1}; gives T_RL for the reciprocity pin.
 * If g_state/P_state are non-NULL the sweep stops after `stop_after` slices have been
 * processed (1..L) and returns g_i and P_i of the last processed slice.
 * ---------------------------------------------------------------------------------------- */
static int sweep(int M, int L, const double *onsite, const uint8_t *vac, double t, double E, double eta,
                 int direction, int lead_method, int stop_after, double *T_out, double *imtrace_out,
                 cplx *g_state, cplx *P_state, int *iters_out)
{
    size_t MM = (size_t)M * M;
    cplx z = c_make(E, eta);
    cplx *buf = (cplx *)malloc(sizeof(cplx) * MM * 9);
    double *mp = (double *)malloc(sizeof(double) * (size_t)M);
    if (!buf || !mp) { free(buf); free(mp); return ORC_ENOMEM; }
    cplx *SigL = buf, *SigR = buf + MM, *A = buf + 2 * MM, *g = buf + 3 * MM, *gprev = buf + 4 * MM;
    cplx *P = buf + 5 * MM, *Pprev = buf + 6 * MM, *H = buf + 7 * MM, *Gm = buf + 8 * MM;
    int itL = 0, itR = 0;
    int rc = lead_self_energy(M, L, vac, t, z, -1, lead_method, SigL, &itL);
    if (rc == ORC_OK) rc = lead_self_energy(M, L, vac, t, z, +1, lead_method, SigR, &itR);
    if (iters_out) { iters_out[0] = itL; iters_out[1] = itR; }
    if (rc != ORC_OK) { free(buf); free(mp); return rc; }
    /* In the mirror sweep the first slice is L-1 (carrying Sigma_R) and the last is 0. */
    const cplx *SigFirst = direction == 0 ? SigL : SigR;
    const cplx *SigLast = direction == 0 ? SigR : SigL;
    int nsteps = (stop_after > 0 && stop_after < L) ? stop_after : L;
    for (int s = 0; s < nsteps; s++) {
        int i = direction == 0 ? s : L - 1 - s;            /* slice being added */
        slice_hamiltonian(M, L, onsite, vac, i, t, H);
        for (size_t k = 0; k < MM; k++) A[k] = c_make(-H[k].re, -H[k].im);
        for (int d = 0; d < M; d++) A[(size_t)d * M + d] = c_add(A[(size_t)d * M + d], z);
        if (s == 0) for (size_t k = 0; k < MM; k++) A[k] = c_sub(A[k], SigFirst[k]);
        if (s == L - 1) for (size_t k = 0; k < MM; k++) A[k] = c_sub(A[k], SigLast[k]);
        if (s > 0) {
            /* bond between the new slice i and the previous one (i-1 or i+1) */
            bond_mask(M, L, vac, direction == 0 ? i - 1 : i, mp);
            /* Sigma = V g_prev V = t^2 m' (.) g_prev (.) m'  (Eq. 4 with the direct form, Q3) */
            for (int r = 0; r < M; r++)
                for (int c = 0; c < M; c++) {
                    cplx sig = c_scale(gprev[(size_t)r * M + c], (t * mp[r]) * (t * mp[c]));
                    A[(size_t)r * M + c] = c_sub(A[(size_t)r * M + c], sig);
                }
        }
        rc = mat_inverse(M, A, g);                          /* G_ii, Eq. 4 */
        if (rc != ORC_OK) break;
        if (s == 0) {
            memcpy(P, g, sizeof(cplx) * MM);                /* P_0 = g_0 */
        } else {
            /* P_i = g_i V P_{i-1}: V = t diag(m') scales the columns of g_i (Eq. 5) */
            for (int r = 0; r < M; r++)
                for (int c = 0; c < M; c++) Gm[(size_t)r * M + c] = c_scale(g[(size_t)r * M + c], t * mp[c]);
            mat_mul(M, Gm, Pprev, P);
        }
        memcpy(gprev, g, sizeof(cplx) * MM);
        memcpy(Pprev, P, sizeof(cplx) * MM);
    }
    if (rc == ORC_OK && g_state && P_state) {
        memcpy(g_state, gprev, sizeof(cplx) * MM);
        memcpy(P_state, Pprev, sizeof(cplx) * MM);
    }
    if (rc == ORC_OK && nsteps == L && T_out) {
        /* O6: Gamma = i (Sigma - Sigma^dagger); T = Re Tr[Gamma_first P^dagger Gamma_last P] (Eq. 2) */
        cplx *GamF = A, *GamL = H, *X = g, *Y = Gm;
        for (int r = 0; r < M; r++)
            for (int c = 0; c < M; c++) {
                cplx a = SigFirst[(size_t)r * M + c], b = SigFirst[(size_t)c * M + r];
                cplx d = c_make(a.re - b.re, a.im + b.im);              /* Sigma - Sigma^dagger */
                GamF[(size_t)r * M + c] = c_make(-d.im, d.re);          /* times i */
                a = SigLast[(size_t)r * M + c]; b = SigLast[(size_t)c * M + r];
                d = c_make(a.re - b.re, a.im + b.im);
                GamL[(size_t)r * M + c] = c_make(-d.im, d.re);
            }
        mat_mul(M, GamL, Pprev, X);                         /* Gamma_R P */
        for (int r = 0; r < M; r++)                         /* P^dagger */
            for (int c = 0; c < M; c++) Y[(size_t)r * M + c] = c_make(Pprev[(size_t)c * M + r].re, -Pprev[(size_t)c * M + r].im);
        mat_mul(M, Y, X, P);                                /* P^dagger Gamma_R P */
        mat_mul(M, GamF, P, X);                             /* Gamma_L P^dagger Gamma_R P */
        cplx tr = c_make(0, 0);
        for (int d = 0; d < M; d++) tr = c_add(tr, X[(size_t)d * M + d]);
        *T_out = tr.re;
        if (imtrace_out) *imtrace_out = tr.im;
    }
    free(buf); free(mp);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O7. Brute force: assemble the whole (M L) x (M L) matrix z - H - Sigma_L (+) Sigma_R,
 * invert it with the same naive LU, read block (L-1, 0) [and (0, L-1)], apply Eq. 2.
 * Only for tiny ribbons (M*L <~ 1000).
 * ---------------------------------------------------------------------------------------- */
static int brute(int M, int L, const double *onsite, const uint8_t *vac, double t, double E, double eta,
                 int lead_method, double *T_LR, double *T_RL)
{
    size_t MM = (size_t)M * M;
    int N = M * L;
    size_t NN = (size_t)N * N;
    cplx z = c_make(E, eta);
    cplx *A = (cplx *)malloc(sizeof(cplx) * NN), *G = (cplx *)malloc(sizeof(cplx) * NN);
    cplx *buf = (cplx *)malloc(sizeof(cplx) * MM * 8);
    double *mp = (double *)malloc(sizeof(double) * (size_t)M);
    if (!A || !G || !buf || !mp) { free(A); free(G); free(buf); free(mp); return ORC_ENOMEM; }
    cplx *SigL = buf, *SigR = buf + MM, *H = buf + 2 * MM, *GamL = buf + 3 * MM, *GamR = buf + 4 * MM;
    cplx *P = buf + 5 * MM, *X = buf + 6 * MM, *Y = buf + 7 * MM;
    int rc = lead_self_energy(M, L, vac, t, z, -1, lead_method, SigL, NULL);
    if (rc == ORC_OK) rc = lead_self_energy(M, L, vac, t, z, +1, lead_method, SigR, NULL);
    if (rc == ORC_OK) {
        for (size_t k = 0; k < NN; k++) A[k] = c_make(0, 0);
        for (int i = 0; i < L; i++) {
            slice_hamiltonian(M, L, onsite, vac, i, t, H);
            for (int r = 0; r < M; r++)
                for (int c = 0; c < M; c++) {
                    cplx v = c_make(-H[(size_t)r * M + c].re, 0.0);
                    if (r == c) v = c_add(v, z);
                    if (i == 0) v = c_sub(v, SigL[(size_t)r * M + c]);
                    if (i == L - 1) v = c_sub(v, SigR[(size_t)r * M + c]);
                    A[(size_t)(i * M + r) * N + (i * M + c)] = v;
                }
            if (i + 1 < L) {
                bond_mask(M, L, vac, i, mp);
                for (int j = 0; j < M; j++) {
                    A[(size_t)(i * M + j) * N + ((i + 1) * M + j)] = c_make(-t * mp[j], 0.0);
                    A[(size_t)((i + 1) * M + j) * N + (i * M + j)] = c_make(-t * mp[j], 0.0);
                }
            }
        }
        rc = mat_inverse(N, A, G);
    }
    if (rc == ORC_OK) {
        for (int r = 0; r < M; r++)
            for (int c = 0; c < M; c++) {
                cplx a = SigL[(size_t)r * M + c], b = SigL[(size_t)c * M + r];
                cplx d = c_make(a.re - b.re, a.im + b.im);
                GamL[(size_t)r * M + c] = c_make(-d.im, d.re);
                a = SigR[(size_t)r * M + c]; b = SigR[(size_t)c * M + r];
                d = c_make(a.re - b.re, a.im + b.im);
                GamR[(size_t)r * M + c] = c_make(-d.im, d.re);
            }
        for (int pass = 0; pass < 2; pass++) {
            /* pass 0: P = G_{L-1,0}, T = Tr[Gam_L P^+ Gam_R P]; pass 1: P = G_{0,L-1}, leads swapped */
            int rb = pass == 0 ? L - 1 : 0, cb = pass == 0 ? 0 : L - 1;
            const cplx *G1 = pass == 0 ? GamL : GamR, *G2 = pass == 0 ? GamR : GamL;
            for (int r = 0; r < M; r++)
                for (int c = 0; c < M; c++) P[(size_t)r * M + c] = G[(size_t)(rb * M + r) * N + (cb * M + c)];
            mat_mul(M, G2, P, X);
            for (int r = 0; r < M; r++)
                for (int c = 0; c < M; c++) Y[(size_t)r * M + c] = c_make(P[(size_t)c * M + r].re, -P[(size_t)c * M + r].im);
            mat_mul(M, Y, X, H);
            mat_mul(M, G1, H, X);
            double tr = 0.0;
            for (int d = 0; d < M; d++) tr += X[(size_t)d * M + d].re;
            if (pass == 0) { if (T_LR) *T_LR = tr; } else { if (T_RL) *T_RL = tr; }
        }
    }
    free(A); free(G); free(buf); free(mp);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O9. Local density of states of the connected device.
 * PAPER.md:37 "Knowledge of the Green's function allows one to compute any desired quantity, e.g.
 * charge density"; PAPER.md:61 (step 5: the Green's functions of the whole region).  Definition:
 *   LDOS(i, j; E) = -(1/pi) Im G_ii[j][j],   G = (z - H_device - Sigma_L (+) 0 (+) Sigma_R)^-1  (Eq. 1)
 * computed by the textbook two-pass recursion for the diagonal blocks (Dyson's equation, Eq. 3,
 * applied from the right after the left-to-right sweep of Eq. 4):
 *   forward   g_i = (z - H_i - V g_{i-1} V [- Sigma_L at 0] [- Sigma_R at L-1])^-1, all g_i kept
 *   backward  G_{L-1,L-1} = g_{L-1};   G_ii = g_i + g_i V G_{i+1,i+1} V g_i,  V = t diag(m'_i)
 * The brute-force pin (the definition itself, by numpy on a matrix the test assembles) is in
 * tests/test_oracle_pins.py.  ldos_out[L][M].
 * ---------------------------------------------------------------------------------------- */
static int ldos_sweep(int M, int L, const double *onsite, const uint8_t *vac, double t, double E, double eta,
                      int lead_method, double *ldos_out)
{
    const double pi = 3.14159265358979323846;
    size_t MM = (size_t)M * M;
    cplx z = c_make(E, eta);
    cplx *gall = (cplx *)malloc(sizeof(cplx) * MM * (size_t)L);
    cplx *buf = (cplx *)malloc(sizeof(cplx) * MM * 7);
    double *mp = (double *)malloc(sizeof(double) * (size_t)M);
    if (!gall || !buf || !mp) { free(gall); free(buf); free(mp); return ORC_ENOMEM; }
    cplx *SigL = buf, *SigR = buf + MM, *A = buf + 2 * MM, *H = buf + 3 * MM, *G = buf + 4 * MM, *X = buf + 5 * MM, *Y = buf + 6 * MM;
    int rc = lead_self_energy(M, L, vac, t, z, -1, lead_method, SigL, NULL);
    if (rc == ORC_OK) rc = lead_self_energy(M, L, vac, t, z, +1, lead_method, SigR, NULL);
    for (int i = 0; i < L && rc == ORC_OK; i++) {
        slice_hamiltonian(M, L, onsite, vac, i, t, H);
        for (size_t k = 0; k < MM; k++) A[k] = c_make(-H[k].re, -H[k].im);
        for (int d = 0; d < M; d++) A[(size_t)d * M + d] = c_add(A[(size_t)d * M + d], z);
        if (i == 0) for (size_t k = 0; k < MM; k++) A[k] = c_sub(A[k], SigL[k]);
        if (i == L - 1) for (size_t k = 0; k < MM; k++) A[k] = c_sub(A[k], SigR[k]);
        if (i > 0) {
            bond_mask(M, L, vac, i - 1, mp);
            const cplx *gp = gall + (size_t)(i - 1) * MM;
            for (int r = 0; r < M; r++)
                for (int c = 0; c < M; c++)
                    A[(size_t)r * M + c] = c_sub(A[(size_t)r * M + c], c_scale(gp[(size_t)r * M + c], (t * mp[r]) * (t * mp[c])));
        }
        rc = mat_inverse(M, A, gall + (size_t)i * MM);
    }
    if (rc == ORC_OK) {
        memcpy(G, gall + (size_t)(L - 1) * MM, sizeof(cplx) * MM);
        for (int i = L - 1; i >= 0; i--) {
            if (i < L - 1) {
                const cplx *gi = gall + (size_t)i * MM;
                bond_mask(M, L, vac, i, mp);
                for (int r = 0; r < M; r++)                       /* V G_{i+1,i+1} V */
                    for (int c = 0; c < M; c++) X[(size_t)r * M + c] = c_scale(G[(size_t)r * M + c], (t * mp[r]) * (t * mp[c]));
                mat_mul(M, gi, X, Y);                               /* g_i V G V */
                mat_mul(M, Y, gi, X);                               /* g_i V G V g_i */
                for (size_t k = 0; k < MM; k++) G[k] = c_add(gi[k], X[k]);
            }
            for (int j = 0; j < M; j++) ldos_out[(size_t)i * M + j] = -G[(size_t)j * M + j].im / pi;
        }
    }
    free(gall); free(buf); free(mp);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O10. The paper's own form of the recursion, in double or in IEEE single precision
 * (SURVEY.md 8(c) "Precision finding"; Eq. 4, Eq. 5).
 *   G0_j  = (z - H_j [- Sigma_L at j = 0] [- Sigma_R at j = L-1])^-1      Green's function of the isolated slice
 *   G_jj  = (1 - G0_j V G_{j-1,j-1} V)^-1 G0_j                             Eq. 4 (Sigma^l, Sigma^r of the paper = the hopping V)
 *   G_j0  = G_jj V G_{j-1,0}                                               Eq. 5 in the column form (reading Q4)
 * Algebraically the same as the direct form of sweep(); numerically not: G0_j is ill-conditioned whenever E is near a
 * level of the isolated slice.  use_float = 1 runs every matrix operation of the sweep and the trace in single precision
 * (own float LU and matmul below); the lead self-energies are computed in double and rounded (reading Q17: the paper
 * computed them on the CPU).  This reproduces the paper's single-precision finding on the CPU; it is not compared with
 * the CUDA path, whose complex64 sweep uses the direct form.
 * ---------------------------------------------------------------------------------------- */
typedef struct { float re, im; } cplxf;
static inline cplxf f_make(float re, float im) { cplxf r; r.re = re; r.im = im; return r; }
static inline cplxf f_add(cplxf a, cplxf b) { return f_make(a.re + b.re, a.im + b.im); }
static inline cplxf f_sub(cplxf a, cplxf b) { return f_make(a.re - b.re, a.im - b.im); }
static inline cplxf f_mul(cplxf a, cplxf b) { return f_make(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
static inline cplxf f_div(cplxf a, cplxf b)
{
    if (fabsf(b.re) >= fabsf(b.im)) {
        float r = b.im / b.re, d = b.re + b.im * r;
        return f_make((a.re + a.im * r) / d, (a.im - a.re * r) / d);
    } else {
        float r = b.re / b.im, d = b.re * r + b.im;
        return f_make((a.re * r + a.im) / d, (a.im * r - a.re) / d);
    }
}

static void mat_mul_f(int n, const cplxf *A, const cplxf *B, cplxf *C)
{
    for (int i = 0; i < n; i++) {
        cplxf *Ci = C + (size_t)i * n;
        for (int j = 0; j < n; j++) Ci[j] = f_make(0.f, 0.f);
        for (int k = 0; k < n; k++) {
            cplxf a = A[(size_t)i * n + k];
            const cplxf *Bk = B + (size_t)k * n;
            for (int j = 0; j < n; j++) Ci[j] = f_add(Ci[j], f_mul(a, Bk[j]));
        }
    }
}

/* the LU of mat_inverse, in single precision (the paper's CGESV) */
static int mat_inverse_f(int n, const cplxf *A, cplxf *Ainv)
{
    cplxf *LU = (cplxf *)malloc(sizeof(cplxf) * (size_t)n * n);
    int *perm = (int *)malloc(sizeof(int) * (size_t)n);
    cplxf *y = (cplxf *)malloc(sizeof(cplxf) * (size_t)n);
    if (!LU || !perm || !y) { free(LU); free(perm); free(y); return ORC_ENOMEM; }
    memcpy(LU, A, sizeof(cplxf) * (size_t)n * n);
    for (int i = 0; i < n; i++) perm[i] = i;
    int rc = ORC_OK;
    for (int k = 0; k < n; k++) {
        int p = k;
        float best = LU[(size_t)k * n + k].re * LU[(size_t)k * n + k].re + LU[(size_t)k * n + k].im * LU[(size_t)k * n + k].im;
        for (int i = k + 1; i < n; i++) {
            cplxf x = LU[(size_t)i * n + k];
            float v = x.re * x.re + x.im * x.im;
            if (v > best) { best = v; p = i; }
        }
        if (!(best > 0.f) || !isfinite(best)) { rc = ORC_ESINGULAR; break; }
        if (p != k) {
            for (int j = 0; j < n; j++) { cplxf tmp = LU[(size_t)k * n + j]; LU[(size_t)k * n + j] = LU[(size_t)p * n + j]; LU[(size_t)p * n + j] = tmp; }
            int tp = perm[k]; perm[k] = perm[p]; perm[p] = tp;
        }
        cplxf piv = LU[(size_t)k * n + k];
        for (int i = k + 1; i < n; i++) {
            cplxf f = f_div(LU[(size_t)i * n + k], piv);
            LU[(size_t)i * n + k] = f;
            cplxf *Li = LU + (size_t)i * n;
            const cplxf *Lk = LU + (size_t)k * n;
            for (int j = k + 1; j < n; j++) Li[j] = f_sub(Li[j], f_mul(f, Lk[j]));
        }
    }
    if (rc == ORC_OK) {
        for (int c = 0; c < n; c++) {
            for (int i = 0; i < n; i++) {
                cplxf sacc = (perm[i] == c) ? f_make(1.f, 0.f) : f_make(0.f, 0.f);
                const cplxf *Li = LU + (size_t)i * n;
                for (int j = 0; j < i; j++) sacc = f_sub(sacc, f_mul(Li[j], y[j]));
                y[i] = sacc;
            }
            for (int i = n - 1; i >= 0; i--) {
                cplxf sacc = y[i];
                const cplxf *Ui = LU + (size_t)i * n;
                for (int j = i + 1; j < n; j++) sacc = f_sub(sacc, f_mul(Ui[j], y[j]));
                y[i] = f_div(sacc, Ui[i]);
            }
            for (int i = 0; i < n; i++) Ainv[(size_t)i * n + c] = y[i];
        }
    }
    free(LU); free(perm); free(y);
    return rc;
}

/* One body for the two precisions: CT = complex type, RT = real type, and its helpers. */
#define ORC_EQ4_SWEEP(NAME, CT, RT, MK, ADD, SUB, MATMUL, MATINV)                                                          \
static int NAME(int M, int L, const double *onsite, const uint8_t *vac, double t, double E, double eta, int lead_method,  \
                double *T_out)                                                                                             \
{                                                                                                                          \
    size_t MM = (size_t)M * M;                                                                                             \
    cplx z = c_make(E, eta);                                                                                               \
    cplx *SigL = (cplx *)malloc(sizeof(cplx) * MM * 3), *SigR = SigL ? SigL + MM : NULL, *H = SigL ? SigL + 2 * MM : NULL;   \
    CT *buf = (CT *)malloc(sizeof(CT) * MM * 8);                                                                           \
    double *mp = (double *)malloc(sizeof(double) * (size_t)M);                                                             \
    if (!SigL || !buf || !mp) { free(SigL); free(buf); free(mp); return ORC_ENOMEM; }                                      \
    CT *A = buf, *G0 = buf + MM, *g = buf + 2 * MM, *gprev = buf + 3 * MM, *P = buf + 4 * MM, *Pprev = buf + 5 * MM,       \
       *X = buf + 6 * MM, *Y = buf + 7 * MM;                                                                               \
    int rc = lead_self_energy(M, L, vac, t, z, -1, lead_method, SigL, NULL);                                               \
    if (rc == ORC_OK) rc = lead_self_energy(M, L, vac, t, z, +1, lead_method, SigR, NULL);                                 \
    for (int i = 0; i < L && rc == ORC_OK; i++) {                                                                          \
        slice_hamiltonian(M, L, onsite, vac, i, t, H);                                                                     \
        for (size_t k = 0; k < MM; k++) {                       /* z - H_i - lead self-energy, formed in double, rounded */ \
            cplx v = c_make(-H[k].re, -H[k].im);                                                                           \
            if (k / M == k % M) v = c_add(v, z);                                                                           \
            if (i == 0) v = c_sub(v, SigL[k]);                                                                             \
            if (i == L - 1) v = c_sub(v, SigR[k]);                                                                         \
            A[k] = MK((RT)v.re, (RT)v.im);                                                                                 \
        }                                                                                                                  \
        rc = MATINV(M, A, G0);                                  /* G0_j of the isolated slice */                           \
        if (rc != ORC_OK) break;                                                                                           \
        if (i == 0) {                                                                                                      \
            memcpy(g, G0, sizeof(CT) * MM);                                                                                \
            memcpy(P, g, sizeof(CT) * MM);                                                                                 \
        } else {                                                                                                           \
            bond_mask(M, L, vac, i - 1, mp);                                                                               \
            for (int r = 0; r < M; r++)                         /* X = V G_{j-1,j-1} V */                                  \
                for (int c = 0; c < M; c++) {                                                                              \
                    RT sc = (RT)((t * mp[r]) * (t * mp[c]));                                                               \
                    X[(size_t)r * M + c] = MK(gprev[(size_t)r * M + c].re * sc, gprev[(size_t)r * M + c].im * sc);         \
                }                                                                                                          \
            MATMUL(M, G0, X, Y);                                /* G0 V G V */                                             \
            for (size_t k = 0; k < MM; k++) Y[k] = MK(-Y[k].re, -Y[k].im);                                                 \
            for (int d = 0; d < M; d++) Y[(size_t)d * M + d] = ADD(Y[(size_t)d * M + d], MK((RT)1, (RT)0));                \
            rc = MATINV(M, Y, X);                               /* (1 - G0 V G V)^-1 */                                    \
            if (rc != ORC_OK) break;                                                                                       \
            MATMUL(M, X, G0, g);                                /* Eq. 4 */                                                \
            for (int r = 0; r < M; r++)                                                                                    \
                for (int c = 0; c < M; c++) {                                                                              \
                    RT sc = (RT)(t * mp[c]);                                                                               \
                    X[(size_t)r * M + c] = MK(g[(size_t)r * M + c].re * sc, g[(size_t)r * M + c].im * sc);                 \
                }                                                                                                          \
            MATMUL(M, X, Pprev, P);                             /* Eq. 5 */                                                \
        }                                                                                                                  \
        memcpy(gprev, g, sizeof(CT) * MM);                                                                                 \
        memcpy(Pprev, P, sizeof(CT) * MM);                                                                                 \
    }                                                                                                                      \
    if (rc == ORC_OK) {                                         /* Eq. 2 in the sweep's precision */                       \
        CT *GamL = A, *GamR = G0;                                                                                          \
        for (int r = 0; r < M; r++)                                                                                        \
            for (int c = 0; c < M; c++) {                                                                                  \
                cplx a = SigL[(size_t)r * M + c], b = SigL[(size_t)c * M + r];                                             \
                GamL[(size_t)r * M + c] = MK((RT)(-(a.im + b.im)), (RT)(a.re - b.re));                                     \
                a = SigR[(size_t)r * M + c]; b = SigR[(size_t)c * M + r];                                                  \
                GamR[(size_t)r * M + c] = MK((RT)(-(a.im + b.im)), (RT)(a.re - b.re));                                     \
            }                                                                                                              \
        MATMUL(M, GamR, Pprev, X);                                                                                         \
        for (int r = 0; r < M; r++)                                                                                        \
            for (int c = 0; c < M; c++) Y[(size_t)r * M + c] = MK(Pprev[(size_t)c * M + r].re, -Pprev[(size_t)c * M + r].im); \
        MATMUL(M, Y, X, P);                                                                                                \
        MATMUL(M, GamL, P, X);                                                                                             \
        double tr = 0.0;                                                                                                   \
        for (int d = 0; d < M; d++) tr += (double)X[(size_t)d * M + d].re;                                                 \
        *T_out = tr;                                                                                                       \
    }                                                                                                                      \
    free(SigL); free(buf); free(mp);                                                                                       \
    return rc;                                                                                                             \
}

ORC_EQ4_SWEEP(sweep_eq4_d, cplx, double, c_make, c_add, c_sub, mat_mul, mat_inverse)
ORC_EQ4_SWEEP(sweep_eq4_f, cplxf, float, f_make, f_add, f_sub, mat_mul_f, mat_inverse_f)

/* ==========================================================================================
 * Exported C ABI of the oracle (loaded through ctypes by oracle/rgf_oracle.py).
 * Complex arrays: interleaved doubles, row-major.
 * ======================================================================================== */

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int orc_inverse(int n, const double *A, double *Ainv)
{
    if (n < 1 || !A || !Ainv) return ORC_EINVAL;
    return mat_inverse(n, (const cplx *)A, (cplx *)Ainv);
}

int orc_matmul(int n, const double *A, const double *B, double *C)
{
    if (n < 1 || !A || !B || !C) return ORC_EINVAL;
    mat_mul(n, (const cplx *)A, (const cplx *)B, (cplx *)C);
    return ORC_OK;
}

/* g_out[M][M]: surface Green's function of the clean lead (side +1 right / -1 left). */
int orc_lead_surface(int M, int L, double t, double E, double eta, int side, int method, double *g_out, int *iters)
{
    if (M < 2 || L < 1 || !(eta > 0.0) || (side != 1 && side != -1) || !g_out) return ORC_EINVAL;
    return lead_surface(M, L, t, c_make(E, eta), side, method, (cplx *)g_out, iters);
}

/* Sigma_out[M][M]: lead self-energy on the device's end slice, vacancy-aware. */
int orc_lead_self_energy(int M, int L, const uint8_t *vac, double t, double E, double eta, int side, int method,
                         double *Sigma_out, int *iters)
{
    if (M < 2 || L < 1 || !(eta > 0.0) || (side != 1 && side != -1) || !Sigma_out) return ORC_EINVAL;
    return lead_self_energy(M, L, vac, t, c_make(E, eta), side, method, (cplx *)Sigma_out, iters);
}

/* T(E) for one energy.  direction 0 = left-to-right (T_LR), 1 = mirror sweep (T_RL). */
int orc_transmission(int M, int L, const double *onsite, const uint8_t *vac, double t, double E, double eta,
                     int direction, int lead_method, double *T_out, double *imtrace_out, int *iters)
{
    if (M < 2 || L < 1 || !(eta > 0.0) || !onsite || !T_out) return ORC_EINVAL;
    return sweep(M, L, onsite, vac, t, E, eta, direction, lead_method, 0, T_out, imtrace_out, NULL, NULL, iters);
}

/* State after `nslices` slices (1..L) of the left-to-right sweep: g = G_ii, P = G_{i,0}, i = nslices-1. */
int orc_sweep_state(int M, int L, const double *onsite, const uint8_t *vac, double t, double E, double eta,
                    int lead_method, int nslices, double *g_out, double *P_out)
{
    if (M < 2 || L < 1 || !(eta > 0.0) || !onsite || nslices < 1 || nslices > L || !g_out || !P_out) return ORC_EINVAL;
    return sweep(M, L, onsite, vac, t, E, eta, 0, lead_method, nslices, NULL, NULL, (cplx *)g_out, (cplx *)P_out, NULL);
}

/* Batch over energies, OpenMP over energies only (nthreads <= 0: all cores).  status[k] gets
 * the per-energy return code; a failed energy gets T = NaN.  Returns the first non-zero code. */
int orc_transmission_batch(int M, int L, const double *onsite, const uint8_t *vac, double t, const double *energies,
                           int n_E, double eta, int lead_method, int nthreads, double *T_out, int *status)
{
    if (M < 2 || L < 1 || n_E < 1 || !(eta > 0.0) || !onsite || !energies || !T_out) return ORC_EINVAL;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    int first = ORC_OK;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int k = 0; k < n_E; k++) {
        double T = NAN;
        int rc = sweep(M, L, onsite, vac, t, energies[k], eta, 0, lead_method, 0, &T, NULL, NULL, NULL, NULL);
        T_out[k] = (rc == ORC_OK) ? T : NAN;
        if (status) status[k] = rc;
        if (rc != ORC_OK) {
#pragma omp critical
            { if (first == ORC_OK) first = rc; }
        }
    }
    return first;
}

int orc_transmission_brute(int M, int L, const double *onsite, const uint8_t *vac, double t, double E, double eta,
                           int lead_method, double *T_LR, double *T_RL)
{
    if (M < 2 || L < 1 || !(eta > 0.0) || !onsite) return ORC_EINVAL;
    if ((long)M * L > 4096) return ORC_EINVAL;
    return brute(M, L, onsite, vac, t, E, eta, lead_method, T_LR, T_RL);
}

/* ldos_out[n_E][L][M] = -(1/pi) Im G_ii[j][j] of the connected device, OpenMP over energies. */
int orc_ldos_batch(int M, int L, const double *onsite, const uint8_t *vac, double t, const double *energies, int n_E,
                   double eta, int lead_method, int nthreads, double *ldos_out)
{
    if (M < 2 || L < 1 || n_E < 1 || !(eta > 0.0) || !onsite || !energies || !ldos_out) return ORC_EINVAL;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    int first = ORC_OK;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int k = 0; k < n_E; k++) {
        int rc = ldos_sweep(M, L, onsite, vac, t, energies[k], eta, lead_method, ldos_out + (size_t)k * L * M);
        if (rc != ORC_OK) {
#pragma omp critical
            { if (first == ORC_OK) first = rc; }
        }
    }
    return first;
}

/* T(E) by the paper's Eq. 4 form (O10), in double (use_float = 0) or IEEE single precision (1); OpenMP over energies. */
int orc_transmission_eq4_batch(int M, int L, const double *onsite, const uint8_t *vac, double t, const double *energies, int n_E,
                               double eta, int use_float, int lead_method, int nthreads, double *T_out, int *status)
{
    if (M < 2 || L < 1 || n_E < 1 || !(eta > 0.0) || !onsite || !energies || !T_out) return ORC_EINVAL;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    int first = ORC_OK;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int k = 0; k < n_E; k++) {
        double T = NAN;
        int rc = use_float ? sweep_eq4_f(M, L, onsite, vac, t, energies[k], eta, lead_method, &T)
                           : sweep_eq4_d(M, L, onsite, vac, t, energies[k], eta, lead_method, &T);
        T_out[k] = (rc == ORC_OK) ? T : NAN;
        if (status) status[k] = rc;
        if (rc != ORC_OK) {
#pragma omp critical
            { if (first == ORC_OK) first = rc; }
        }
    }
    return first;
}
