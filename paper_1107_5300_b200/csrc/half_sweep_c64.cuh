// half_sweep_c64.cuh -- the complex64 sweep (BASELINE.json:configs[3], the paper's single-precision study,
// PAPER.md:82) for M <= 256: the half-slice recursion of half_kernels.cuh with every step of the sweep
// (assembly, inverse, propagator product) in IEEE single precision on the FP32 FFMA pipe.
//
// Units: the kernel works in units of the hopping, A~ = A / t, g~ = t g: then every coupling is exactly 1 (Sigma~ = m g~ m,
// P <- g~ (m P)), so the same hopping enters the self-energy and the propagation bit for bit.  (With t^2 rounded for
// one and t for the other the mismatch float(t^2) / float(t)^2 - 1 = -4e-8 acts as a gain per half-step and T drifts
// by 1.7e-4 T over 4000 half-steps.)  The propagator carries one overall factor t, divided out in double at the end.
//
// Reading R13: the lead surface Green's functions are computed in complex128 and rounded; (E - eps_j)
// is formed in double and rounded; the Gamma trace runs in double on the rounded propagator.  Everything between
// is float.  TF32 tensor cores are not used: their 10-bit mantissa cannot hold 1e-3 over thousands of slices.
//
// One CTA (512 threads) owns one (device, energy) pair for the whole sweep.  The n x n matrix of a half-step
// lives in REGISTERS during the elimination (thread (w, l) = (warp, lane) owns rows w + 16 i, columns l + 32 j:
// 8 x 4 elements), g of the previous half-step in shared memory, only the propagator streams through L2:
//     assembly   A <- z - eps - C g_prev C^T [- Sigma]          registers <- shared memory
//     inverse    unblocked Gauss-Jordan with partial pivoting (rows never move), 2 barriers per pivot
//     g          scattered to shared memory in true order       g[k][p_c] = X[p_k][c]
//     propagator P <- g (C P_prev), 32-column tiles of C P_prev staged in shared memory, FFMA register tiles
#pragma once
#include "half_kernels.cuh"
#include "rgf_common.cuh"

namespace rgf {

constexpr int HC_NT = 512, HC_NMAX = 128, HC_LDG = HC_NMAX + 1, HC_LDW = 33;

struct HC64Args {
    int M, L, nh, n_E, bz0, nb;
    double eta, t;
    const double *energies, *onsite;
    const uint8_t *bond, *hop;
    const cplx *gL, *gR;              // complex128 lead surface Green's functions [n_E][M][M]
    float2 *P0, *P1;                  // [nb][HC_NMAX * HC_NMAX] propagator ping-pong (ld HC_NMAX)
    int *status;                      // [nb]
    int hs_end;                       // half-steps [0, hs_end)
    cplx *g_out, *P_out;              // complex128 copies of the final g (dense n x n, ld n) and P (ld nh), stride nh*nh
};

struct HC64Smem {
    float2 g[HC_NMAX * HC_LDG];       // g of the previous half-step, true order
    float2 Wt[HC_NMAX * HC_LDW];      // tile of C P_prev
    float2 colk[2][HC_NMAX], prow[2][HC_NMAX];
    float eps_re[HC_NMAX];            // E - eps_j, formed in double, rounded
    short ra[HC_NMAX], rb[HC_NMAX];   // kind B: ra = m'; kind F: lower / upper B neighbour (or -1)
    int perm[HC_NMAX], pinv[HC_NMAX];
    unsigned char used[HC_NMAX];
};

__device__ __forceinline__ float2 c64mul(float2 a, float2 b) { return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x)); }

__global__ void __launch_bounds__(HC_NT, 1) half_sweep_c64_kernel(HC64Args a)
{
    extern __shared__ __align__(16) unsigned char hc_raw[];
    HC64Smem &sm = *reinterpret_cast<HC64Smem *>(hc_raw);
    const int bl = blockIdx.x, tid = threadIdx.x, w = tid >> 5, l = tid & 31;
    const int M = a.M, L = a.L, nc = M / 2;
    const int bz = a.bz0 + bl, d = bz / a.n_E, e = bz % a.n_E;
    const long long MM = (long long)M * M;
    const double E = a.energies[e];
    const float etaf = (float)(a.eta / a.t);          // Im z / t
    float2 *Pb[2] = {a.P0 + (long long)bl * HC_NMAX * HC_NMAX, a.P1 + (long long)bl * HC_NMAX * HC_NMAX};
    const cplx *gl = a.gL + (long long)e * MM, *gr = a.gR + (long long)e * MM;
    int n = 0;
    float2 X[8][4];

    for (int hs = 0; hs < a.hs_end; hs++) {
        const int i = hs >> 1, kind = hs & 1, cur = hs & 1;
        const int par = kind == 0 ? ((i + 1) & 1) : (i & 1);
        n = half_count(M, par);
        const double *eps = a.onsite + ((long long)d * L + i) * M;
        const uint8_t *mk = a.bond + ((long long)d * (L + 1) + i) * M;       // m'_{i-1}
        const uint8_t *mr = a.bond + ((long long)d * (L + 1) + L) * M;       // m'_{L-1}
        const uint8_t *hp = a.hop + ((long long)d * L + i) * M;
        const bool first = hs == 0, last = (kind == 1 && i == L - 1);
        // ---- row tables ----
        if (tid < n) {
            const int r = tid;
            sm.eps_re[r] = (float)((E - eps[2 * r + par]) / a.t);
            if (kind == 0) { sm.ra[r] = mk[2 * r + par] ? 1 : 0; sm.rb[r] = -1; }
            else { sm.ra[r] = (short)half_nbr(r, par, 0, M, hp); sm.rb[r] = (short)half_nbr(r, par, 1, M, hp); }
            sm.used[r] = 0;
        }
        __syncthreads();
        // ---- assembly into registers ----
#pragma unroll
        for (int ii = 0; ii < 8; ii++)
#pragma unroll
            for (int jj = 0; jj < 4; jj++) {
                const int r = w + 16 * ii, c = l + 32 * jj;
                float2 v = make_float2(0.f, 0.f);
                if (r < n && c < n) {
                    if (r == c) v = make_float2(sm.eps_re[r], etaf);
                    float sx = 0.f, sy = 0.f;
                    if (kind == 0) {
                        if (sm.ra[r] && sm.ra[c]) {
                            if (first) { const cplx gg = gl[(long long)(2 * r + par) * M + 2 * c + par]; sx = (float)(a.t * gg.x); sy = (float)(a.t * gg.y); }
                            else { const float2 gg = sm.g[r * HC_LDG + c]; sx = gg.x; sy = gg.y; }
                        }
                    } else {
                        const int ua = sm.ra[r], ub = sm.rb[r], ca = sm.ra[c], cb = sm.rb[c];
                        if (ua >= 0) {
                            if (ca >= 0) { const float2 gg = sm.g[ua * HC_LDG + ca]; sx += gg.x; sy += gg.y; }
                            if (cb >= 0) { const float2 gg = sm.g[ua * HC_LDG + cb]; sx += gg.x; sy += gg.y; }
                        }
                        if (ub >= 0) {
                            if (ca >= 0) { const float2 gg = sm.g[ub * HC_LDG + ca]; sx += gg.x; sy += gg.y; }
                            if (cb >= 0) { const float2 gg = sm.g[ub * HC_LDG + cb]; sx += gg.x; sy += gg.y; }
                        }
                    }
                    v.x -= sx; v.y -= sy;
                    // intra-slice hopping of H_i / t: none inside a half-slice (B and F atoms alternate along the chain)
                    if (last) {
                        const int jr = 2 * r + par, jc = 2 * c + par;
                        if (mr[jr] && mr[jc]) { const cplx gg = gr[(long long)jr * M + jc]; v.x -= (float)(a.t * gg.x); v.y -= (float)(a.t * gg.y); }
                    }
                }
                X[ii][jj] = v;
            }
        __syncthreads();          // everybody has read g_prev
        // ---- Gauss-Jordan with partial pivoting in registers ----
        // Columns are eliminated in a rotated order that changes from half-step to half-step.  In a clean ribbon every slice
        // repeats the same arithmetic on the same numbers, so the rounding errors of a fixed elimination order repeat too
        // and add up coherently: an effective gain or loss per slice, |dT| growing linearly with L (measured on the clean
        // configs[3] ribbon: median 3.0e-4, maximum 1.5e-3 at L = 2000, ten times the disordered ribbon's; carrying the
        // propagator in double or symmetrising g changed nothing).  A different order per half-step gives the same inverse
        // with different roundings, and the errors add like a random walk instead (median 6e-5, maximum 3.2e-4).
        const int shift = (int)(((unsigned)hs * 2654435761u >> 8) % (unsigned)n);
        for (int step = 0; step < n; step++) {
            const int k = (step + shift < n) ? step + shift : step + shift - n;
            const int kb = step & 1, jk = k >> 5;
            if (l == (k & 31)) {
#pragma unroll
                for (int ii = 0; ii < 8; ii++) {
                    float2 v = X[ii][0];
#pragma unroll
                    for (int jj = 1; jj < 4; jj++) if (jj == jk) v = X[ii][jj];
                    sm.colk[kb][w + 16 * ii] = v;
                }
            }
            __syncthreads();
            // every warp finds the pivot itself (same data, same answer): lane handles rows l, l+32, l+64, l+96
            float best = -1.f; int brow = 0;
#pragma unroll
            for (int q = 0; q < 4; q++) {
                const int r = l + 32 * q;
                if (r < n && !sm.used[r]) {
                    const float2 v = sm.colk[kb][r];
                    float m2 = fmaf(v.x, v.x, v.y * v.y);
                    if (!(m2 == m2)) m2 = 3.0e38f;            // NaN: report it
                    if (m2 > best) { best = m2; brow = r; }
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const float ob = __shfl_xor_sync(0xffffffffu, best, o);
                const int orow = __shfl_xor_sync(0xffffffffu, brow, o);
                if (ob > best || (ob == best && orow < brow)) { best = ob; brow = orow; }
            }
            const int p = brow;
            const float2 xp = sm.colk[kb][p];
            const float inv = 1.0f / best;
            const float2 dd = make_float2(xp.x * inv, -xp.y * inv);
            if (w == (p & 15)) {
                const int ip = p >> 4;
#pragma unroll
                for (int jj = 0; jj < 4; jj++) {
                    float2 v = X[0][jj];
#pragma unroll
                    for (int ii = 1; ii < 8; ii++) if (ii == ip) v = X[ii][jj];
                    sm.prow[kb][l + 32 * jj] = c64mul(v, dd);
                }
            }
            __syncthreads();
            if (tid == 0) {          // after the barrier: no warp is still searching with used[]
                if (!(best > 0.f) || !(best < 3.0e38f)) a.status[bl] = 1;
                sm.used[p] = 1; sm.perm[k] = p; sm.pinv[p] = k;
            }
#pragma unroll
            for (int ii = 0; ii < 8; ii++) {
                const int r = w + 16 * ii;
                const bool is_piv = (r == p);
                const float2 xr = sm.colk[kb][r];                 // multiplier of the SCALED pivot row
                const float2 f = c64mul(xr, dd);
#pragma unroll
                for (int jj = 0; jj < 4; jj++) {
                    const int c = l + 32 * jj;
                    const float2 pr = sm.prow[kb][c];
                    float2 v = X[ii][jj];
                    if (c == k) v = is_piv ? dd : make_float2(-f.x, -f.y);
                    else if (is_piv) v = pr;
                    else { v.x = fmaf(-xr.x, pr.x, v.x); v.x = fmaf(xr.y, pr.y, v.x); v.y = fmaf(-xr.x, pr.y, v.y); v.y = fmaf(-xr.y, pr.x, v.y); }
                    X[ii][jj] = v;
                }
            }
        }
        __syncthreads();
        // ---- g[k][p_c] = X[p_k][c] -> shared memory in true order ----
#pragma unroll
        for (int ii = 0; ii < 8; ii++)
#pragma unroll
            for (int jj = 0; jj < 4; jj++) {
                const int r = w + 16 * ii, c = l + 32 * jj;
                if (r < n && c < n) sm.g[sm.pinv[r] * HC_LDG + sm.perm[c]] = X[ii][jj];
            }
        __syncthreads();
        // ---- P_new = g (C P_prev), 32-column tiles ----
        const float2 *Pp = Pb[cur];
        float2 *Pn = Pb[cur ^ 1];
        for (int j0 = 0; j0 < nc; j0 += 32) {
            for (int idx = tid; idx < n * 32; idx += HC_NT) {
                const int m = idx >> 5, jj = idx & 31, j = j0 + jj;
                float2 v = make_float2(0.f, 0.f);
                if (j < nc) {
                    if (first) v = make_float2(m == j ? 1.f : 0.f, 0.f);
                    else if (kind == 0) { if (sm.ra[m]) v = Pp[m * HC_NMAX + j]; }
                    else {
                        const int ua = sm.ra[m], ub = sm.rb[m];
                        float sx = 0.f, sy = 0.f;
                        if (ua >= 0) { const float2 q = Pp[ua * HC_NMAX + j]; sx += q.x; sy += q.y; }
                        if (ub >= 0) { const float2 q = Pp[ub * HC_NMAX + j]; sx += q.x; sy += q.y; }
                        v = make_float2(sx, sy);
                    }
                }
                sm.Wt[m * HC_LDW + jj] = v;
            }
            __syncthreads();
            float2 acc[8];
#pragma unroll
            for (int ii = 0; ii < 8; ii++) acc[ii] = make_float2(0.f, 0.f);
            for (int m = 0; m < n; m++) {
                const float2 wv = sm.Wt[m * HC_LDW + l];
#pragma unroll
                for (int ii = 0; ii < 8; ii++) {
                    const float2 gv = sm.g[(w + 16 * ii) * HC_LDG + m];
                    acc[ii].x = fmaf(gv.x, wv.x, acc[ii].x); acc[ii].x = fmaf(-gv.y, wv.y, acc[ii].x);
                    acc[ii].y = fmaf(gv.x, wv.y, acc[ii].y); acc[ii].y = fmaf(gv.y, wv.x, acc[ii].y);
                }
            }
#pragma unroll
            for (int ii = 0; ii < 8; ii++) {
                const int r = w + 16 * ii;
                if (r < n && j0 + l < nc) Pn[r * HC_NMAX + j0 + l] = acc[ii];
            }
            __syncthreads();
        }
        __threadfence_block();
    }
    // ---- complex128 copies of the final state for the trace / rgf_sweep_state ----
    if (a.hs_end > 0) {
        const long long os = (long long)a.nh * a.nh;
        const float2 *Pf = Pb[a.hs_end & 1];
        if (a.g_out)
            for (int idx = tid; idx < n * n; idx += HC_NT) {
                const float2 v = sm.g[(idx / n) * HC_LDG + idx % n];
                a.g_out[bl * os + idx] = cmake((double)v.x / a.t, (double)v.y / a.t);
            }
        if (a.P_out)
            for (int idx = tid; idx < n * nc; idx += HC_NT) {
                const int k = idx / nc, c = idx % nc;
                const float2 v = Pf[k * HC_NMAX + c];
                if (!(fabsf(v.x) < 3.0e38f) || !(fabsf(v.y) < 3.0e38f)) a.status[bl] = 1;     // overflow / NaN in single precision
                a.P_out[bl * os + (long long)k * a.nh + c] = cmake((double)v.x / a.t, (double)v.y / a.t);
            }
    }
}

}  // namespace rgf
