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
// lives in REGISTERS during the elimination: four threads per row (r = tid / 4, q = tid % 4), thread q holding the working
// columns 4 s + q, s = 0..31, in 32 register slots.  The column being eliminated always sits in slot 0 (static register
// index: no select chains, no spills): after the four pivots of a group the slots rotate by one.  g of the previous half-step
// lives in shared memory, only the propagator streams through L2:
//     assembly   A <- z - eps - C g_prev C^T [- Sigma]          registers <- shared memory
//     inverse    unblocked Gauss-Jordan with partial pivoting (rows never move): integer key + REDUX search, the row's
//                multiplier by a shuffle inside its four threads, 2 barriers per pivot
//     g          scattered to shared memory in true order       g[k][p_c] = X[p_k][c]
//     propagator P <- g (C P_prev), 64-column tiles of C P_prev staged in shared memory, FFMA register tiles (8 rows x 2 columns)
#pragma once
#include "half_kernels.cuh"
#include "rgf_common.cuh"

namespace rgf {

constexpr int HC_NT = 512, HC_NMAX = 128, HC_LDG = HC_NMAX + 1, HC_TW = 64, HC_LDW = HC_TW + 2;

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
    alignas(16) float2 Wt[HC_NMAX * HC_LDW];      // tile of C P_prev (64 columns)
    alignas(16) float2 prow[4 * 34];  // pivot row as it stands (unscaled), thread q's 32 slots at prow[34 q + s] (34: LDS.128 conflict-free)
    alignas(16) unsigned wkey[HC_NT / 32];   // per-warp maximum of the search key (read four at a time)
    float eps_re[HC_NMAX];            // E - eps_j, formed in double, rounded
    short ra[HC_NMAX], rb[HC_NMAX];   // kind B: ra = m'; kind F: lower / upper B neighbour (or -1)
    int perm[HC_NMAX], pinv[HC_NMAX];
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
    const int rr_ = tid >> 2, q = tid & 3, lane = l;       // row of this thread, its column residue, lane
    float2 X[32];

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
        }
        __syncthreads();
        // Columns are eliminated in a rotated order that changes from half-step to half-step: working column c' is true
        // column (c' + shift) mod n.  In a clean ribbon every slice repeats the same arithmetic on the same numbers, so the
        // rounding errors of a fixed elimination order repeat too and add up coherently: an effective gain or loss per slice,
        // |dT| growing linearly with L (measured on the clean configs[3] ribbon: median 3.0e-4, maximum 1.5e-3 at L = 2000,
        // ten times the disordered ribbon's; carrying the propagator in double or symmetrising g changed nothing).  A
        // different order per half-step gives the same inverse with different roundings, and the errors add like a random
        // walk instead (median 6e-5, maximum 3.2e-4).
        const int shift = (int)(((unsigned)hs * 2654435761u >> 8) % (unsigned)n);
        // ---- assembly into registers: slot s <- A[r][(4 s + q + shift) mod n] ----
        {
            const int r = rr_;
            const bool rok = r < n;
            const int ua = rok ? sm.ra[r] : -1, ub = rok ? sm.rb[r] : -1;
            const float er = rok ? sm.eps_re[r] : 0.f;
#pragma unroll
            for (int sl = 0; sl < 32; sl++) {
                const int cw = 4 * sl + q;
                int c = cw + shift; if (c >= n) c -= n;
                float2 v = make_float2(0.f, 0.f);
                if (rok && cw < n) {
                    if (r == c) v = make_float2(er, etaf);
                    float sx = 0.f, sy = 0.f;
                    if (kind == 0) {
                        if (ua && sm.ra[c]) {
                            if (first) { const cplx gg = gl[(long long)(2 * r + par) * M + 2 * c + par]; sx = (float)(a.t * gg.x); sy = (float)(a.t * gg.y); }
                            else { const float2 gg = sm.g[r * HC_LDG + c]; sx = gg.x; sy = gg.y; }
                        }
                    } else {
                        const int ca = sm.ra[c], cb = sm.rb[c];
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
                X[sl] = v;
            }
        }
        __syncthreads();          // everybody has read g_prev
        // ---- Gauss-Jordan with partial pivoting in registers ----
        bool used = !(rr_ < n);
        const int ngroups = (n + 3) >> 2;
#pragma unroll 1
        for (int g4 = 0; g4 < ngroups; g4++) {
#pragma unroll
            for (int qq = 0; qq < 4; qq++) {
                const int cw = 4 * g4 + qq;                 // working column of this step, in slot 0 of the threads q == qq
                if (cw < n) {
                    int k = cw + shift; if (k >= n) k -= n;
                    // search key: top 25 bits of max(|re|, |im|) | (127 - row): unique, names the row, lowest row wins ties
                    const float2 x0 = X[0];
                    const unsigned ure = __float_as_uint(x0.x) & 0x7fffffffu, uim = __float_as_uint(x0.y) & 0x7fffffffu;
                    unsigned key = 0u;
                    if (q == qq) key = (used ? 0u : (max(ure, uim) & 0xffffff80u)) | (unsigned)(127 - rr_);
                    const unsigned wmax = __reduce_max_sync(0xffffffffu, key);
                    if (lane == 0) sm.wkey[w] = wmax;
                    // the row's multiplier (its entry in the working column) for all four threads of the row
                    float2 xr;
                    xr.x = __shfl_sync(0xffffffffu, x0.x, (lane & ~3) | qq);
                    xr.y = __shfl_sync(0xffffffffu, x0.y, (lane & ~3) | qq);
                    __syncthreads();
                    unsigned best = 0u;
#pragma unroll
                    for (int ww = 0; ww < HC_NT / 32; ww += 4) {
                        const uint4 k4 = *reinterpret_cast<const uint4 *>(&sm.wkey[ww]);
                        best = max(max(best, max(k4.x, k4.y)), max(k4.z, k4.w));
                    }
                    const int p = 127 - (int)(best & 127u);
                    const bool is_piv = (rr_ == p);
                    if (is_piv) {
                        // the pivot row publishes itself as it stands; every row scales its own multiplier instead (f = x_r / pivot)
                        float4 *dst = reinterpret_cast<float4 *>(sm.prow + 34 * q);
#pragma unroll
                        for (int sl = 0; sl < 32; sl += 2) dst[sl >> 1] = make_float4(X[sl].x, X[sl].y, X[sl + 1].x, X[sl + 1].y);
                        if (q == qq) {
                            if ((best >> 7) == 0u || best >= 0x7f800000u) a.status[bl] = 1;       // zero / non-finite pivot
                            sm.perm[k] = p; sm.pinv[p] = k;
                        }
                        used = true;
                    }
                    // 1 / pivot from the pivot element, which every thread of the CTA can read after the barrier
                    __syncthreads();
                    const float2 xp = sm.prow[34 * qq];                  // slot 0 of thread qq of the pivot row = the pivot element
                    const float m2 = fmaf(xp.x, xp.x, xp.y * xp.y);
                    const float inv = 1.0f / m2;
                    const float2 dd = make_float2(xp.x * inv, -xp.y * inv);
                    const float2 f = c64mul(xr, dd);                     // multiplier of the unscaled pivot row
                    const float4 *prq = reinterpret_cast<const float4 *>(sm.prow + 34 * q);
                    if ((p >> 3) != w) {
                        // no row of this warp is the pivot row (15 warps of 16): v <- v - f * prow, nothing to select
#pragma unroll
                        for (int sl = 0; sl < 32; sl += 2) {
                            const float4 pr = prq[sl >> 1];
                            float2 v = X[sl], u = X[sl + 1];
                            v.x = fmaf(-f.x, pr.x, v.x); v.x = fmaf(f.y, pr.y, v.x); v.y = fmaf(-f.x, pr.y, v.y); v.y = fmaf(-f.y, pr.x, v.y);
                            u.x = fmaf(-f.x, pr.z, u.x); u.x = fmaf(f.y, pr.w, u.x); u.y = fmaf(-f.x, pr.w, u.y); u.y = fmaf(-f.y, pr.z, u.y);
                            X[sl] = v; X[sl + 1] = u;
                        }
                        if (q == qq) X[0] = make_float2(-f.x, -f.y);
                    } else {
#pragma unroll
                        for (int sl = 0; sl < 32; sl++) {
                            const float2 pr = sm.prow[34 * q + sl];
                            float2 v = X[sl];
                            if (sl == 0 && q == qq) v = is_piv ? dd : make_float2(-f.x, -f.y);
                            else if (is_piv) v = c64mul(pr, dd);
                            else { v.x = fmaf(-f.x, pr.x, v.x); v.x = fmaf(f.y, pr.y, v.x); v.y = fmaf(-f.x, pr.y, v.y); v.y = fmaf(-f.y, pr.x, v.y); }
                            X[sl] = v;
                        }
                    }
                }
            }
            // rotate the slots: the next group's working columns move into slot 0
            const float2 x0 = X[0];
#pragma unroll
            for (int sl = 0; sl < 31; sl++) X[sl] = X[sl + 1];
            X[31] = x0;
        }
        __syncthreads();
        // ---- g[k][p_c] = X[p_k][c] -> shared memory in true order (slot sl holds working slot (ngroups + sl) mod 32) ----
        if (rr_ < n) {
            const int pr_ = sm.pinv[rr_];
#pragma unroll
            for (int sl = 0; sl < 32; sl++) {
                const int cw = 4 * ((ngroups + sl) & 31) + q;
                if (cw < n) {
                    int c = cw + shift; if (c >= n) c -= n;
                    sm.g[pr_ * HC_LDG + sm.perm[c]] = X[sl];
                }
            }
        }
        __syncthreads();
        // ---- P_new = g (C P_prev), 64-column tiles: thread (w, l) takes rows w + 16 i, columns 2 l and 2 l + 1 of the tile ----
        const float2 *Pp = Pb[cur];
        float2 *Pn = Pb[cur ^ 1];
        for (int j0 = 0; j0 < nc; j0 += HC_TW) {
            for (int idx = tid; idx < n * HC_TW; idx += HC_NT) {
                const int m = idx / HC_TW, jj = idx % HC_TW, j = j0 + jj;
                float2 v = make_float2(0.f, 0.f);
                if (j < nc) {
                    if (first) v = make_float2(m == j ? 1.f : 0.f, 0.f);
                    else if (kind == 0) { if (sm.ra[m]) v = Pp[m * HC_NMAX + j]; }
                    else {
                        const int ua = sm.ra[m], ub = sm.rb[m];
                        float sx = 0.f, sy = 0.f;
                        if (ua >= 0) { const float2 qv = Pp[ua * HC_NMAX + j]; sx += qv.x; sy += qv.y; }
                        if (ub >= 0) { const float2 qv = Pp[ub * HC_NMAX + j]; sx += qv.x; sy += qv.y; }
                        v = make_float2(sx, sy);
                    }
                }
                sm.Wt[m * HC_LDW + jj] = v;
            }
            __syncthreads();
            float2 acc[8][2];
#pragma unroll
            for (int ii = 0; ii < 8; ii++) acc[ii][0] = acc[ii][1] = make_float2(0.f, 0.f);
            for (int m = 0; m < n; m++) {
                const float4 wv = *reinterpret_cast<const float4 *>(&sm.Wt[m * HC_LDW + 2 * l]);
#pragma unroll
                for (int ii = 0; ii < 8; ii++) {
                    const float2 gv = sm.g[(w + 16 * ii) * HC_LDG + m];
                    acc[ii][0].x = fmaf(gv.x, wv.x, acc[ii][0].x); acc[ii][0].x = fmaf(-gv.y, wv.y, acc[ii][0].x);
                    acc[ii][0].y = fmaf(gv.x, wv.y, acc[ii][0].y); acc[ii][0].y = fmaf(gv.y, wv.x, acc[ii][0].y);
                    acc[ii][1].x = fmaf(gv.x, wv.z, acc[ii][1].x); acc[ii][1].x = fmaf(-gv.y, wv.w, acc[ii][1].x);
                    acc[ii][1].y = fmaf(gv.x, wv.w, acc[ii][1].y); acc[ii][1].y = fmaf(gv.y, wv.z, acc[ii][1].y);
                }
            }
#pragma unroll
            for (int ii = 0; ii < 8; ii++) {
                const int r = w + 16 * ii, j = j0 + 2 * l;
                if (r < n) {
                    if (j < nc) Pn[r * HC_NMAX + j] = acc[ii][0];
                    if (j + 1 < nc) Pn[r * HC_NMAX + j + 1] = acc[ii][1];
                }
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
