// half_sweep.cuh -- the fused sweep kernel of the half-slice formulation for M <= 256 (n = M/2 <= 128;
// the paper's 30 nm ribbon is M = 244, n = 122).
//
// One CTA owns one (device, energy) pair and runs its half-steps back to back (Eq. 4-5
// on the slicing B_0, F_0, B_1, F_1, ...; half_kernels.cuh states the recursion):
//     A = z - eps - C g_prev C^T  [- Sigma_L/R at the ends]         assembly, O(n^2), staged through smem
//     [ g | P ] = A^-1 [ I | C P_prev ]                            ONE in-place Gauss-Jordan on the augmented matrix
// The propagator columns ride along as extra right-hand sides of the elimination, so inverse (8 n^3)
// and propagator product (8 n^3 real flops) are the same kernel loop: for every panel of 32 columns
//     1. the n x 32 panel is factored in shared memory with partial pivoting (rows never move; thread = row;
//        8-column sub-blocks in registers, the other panel columns by DMMA),
//     2. every other 32-column chunk of [X | W] is updated in place, C += Mult * R on the FP64 tensor
//        pipe (mma.sync m8n8k4 = DMMA.8x8x4), Mult read from the factored panel in shared memory, the
//        32 pivot rows R staged by cp.async, C fragments straight from / to L2.
// Rows are never exchanged: with p_k the pivot row of column k the result sits at
//     g[k][p_c] = X[p_k][c],   P[k][:] = W[p_k][:]
// and the next half-step reads it through the maps perm[k] = p_k, pinv[p_k] = k (no unpermute pass).
// State per matrix in HBM/L2: X (2 buffers), W (2 buffers), perm.  2 CTAs per SM (113 KB of shared
// memory each, <= 128 registers) so that one CTA's latency-bound pivot search overlaps the other's DMMAs.
#pragma once
#include "half_kernels.cuh"
#include "rgf_common.cuh"

namespace rgf {

constexpr int HS_NT = 256, HS_NMAX = 128, HS_B = 32, HS_SB = 8;
constexpr int HS_LDP = HS_B + 4;        // 36: A-fragment reads of the panel conflict-free
constexpr int HS_LDR = HS_B + 2;        // 34: B-fragment reads conflict-free
constexpr int HS_STAGE_ROWS = 36;       // the panel buffer seen as rows of HS_NMAX elements (assembly staging)

struct HSweepArgs {
    int M, L, nh, ldn, n_E, bz0, nb;
    double eta, t;
    const double *energies, *onsite;
    const uint8_t *bond, *hop;
    const cplx *gL, *gR;
    cplx *X0, *X1, *P0, *P1;      // [nb][ldn*ldn] each
    int *perm;                    // [nb][HS_NMAX]
    int *status;                  // [nb]
    int hs_begin, hs_end;         // half-steps [begin, end): hs = 2 i + kind
    long long *prof;              // optional [nb][8] cycle counters of thread 0 per phase (NULL = off)
    cplx *g_out, *P_out;          // after half-step hs_end - 1: g dense n x n (ld n) and P (ld nh), stride nh*nh; may be NULL
};

struct HSmem {
    cplx panel[HS_NMAX * HS_LDP];
    cplx R[2][HS_B * HS_LDR];
    cplx crow[2 * (HS_NT / 32) * HS_SB];
    cplx cinv[2 * (HS_NT / 32)];
    unsigned ckey[2 * (HS_NT / 32)];
    int cidx[2 * (HS_NT / 32)];
    int perm[HS_NMAX], pinv[HS_NMAX], perm_prev[HS_NMAX], pinv_prev[HS_NMAX];
    int prow[HS_B];
    int flag;
};

// per-row tables of the assembly; aliases HSmem::crow while no panel is being factored
struct HSTab {
    double eps[HS_NMAX];
    short ra[HS_NMAX], rb[HS_NMAX], ca[HS_NMAX], cb[HS_NMAX];
};
static_assert(sizeof(HSTab) <= sizeof(cplx) * 2 * (HS_NT / 32) * HS_SB, "HSTab must fit in HSmem::crow");

__device__ __forceinline__ cplx ldcg(const cplx *p)
{
    double2 v = __ldcg(reinterpret_cast<const double2 *>(p));
    return v;
}

// 1 / v for v = |x|^2 > 0: single-precision seed + two Newton steps in FP64 (4 dependent DFMAs instead of
// the ~30 of the IEEE division, which sits on the critical path of every pivot); falls back to the division
// outside the float range.  Relative error ~1e-16, irrelevant for a pivot reciprocal.
__device__ __forceinline__ double hs_rcp(double v)
{
    if (!(v > 1e-30 && v < 1e30)) return 1.0 / v;
    double r = (double)__frcp_rn((float)v);
    double e = fma(-v, r, 1.0);
    r = fma(r, e, r);
    e = fma(-v, r, 1.0);
    return fma(r, e, r);
}

// barrier among the first nthreads threads of the CTA (whole warps); id 1 (0 is __syncthreads)
__device__ __forceinline__ void hs_bar_active(int nthreads) { asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory"); }

// one pivot step on column CC (static) of the thread's 8-column sub-block
template <int CC>
__device__ __forceinline__ void hs_pivot_step(HSmem &sm, cplx (&row)[HS_SB], bool &used, int r, int lane, int warp, int naw,
                                              int kglob, int *status_slot)
{
    constexpr int SB = HS_SB, NW = HS_NT / 32;
    constexpr int pb = (CC & 1) * NW;
    const cplx x = row[CC];
    // 32-bit key: top 24 bits of |x|^2 and 255 - warp (lowest warp / lane wins ties)
    const double v = cabs2(x);
    unsigned hi = used ? 0u : ((unsigned)__double2hiint(v) & 0xffffff00u);
    if (!used && !(v == v)) hi = 0x7ff80000u;
    const unsigned wmax = __reduce_max_sync(0xffffffffu, hi);
    const unsigned ball = __ballot_sync(0xffffffffu, hi == wmax);
    if (lane == __ffs(ball) - 1) {
        sm.ckey[pb + warp] = wmax | (unsigned)(255 - warp);
        sm.cidx[pb + warp] = r;
        const double iv = hs_rcp(v);
        sm.cinv[pb + warp] = cmake(x.x * iv, -x.y * iv);
#pragma unroll
        for (int j = 0; j < SB; j++) sm.crow[(pb + warp) * SB + j] = row[j];
    }
    hs_bar_active(naw * 32);
    unsigned best = sm.ckey[pb];
#pragma unroll
    for (int w = 1; w < NW; w++) if (w < naw) best = max(best, sm.ckey[pb + w]);
    const int pw = 255 - (int)(best & 0xffu);
    const int pr = sm.cidx[pb + pw];
    const cplx d = sm.cinv[pb + pw];
    if (r == pr) {
        if ((best >> 8) == 0u || best >= 0x7ff00000u) *status_slot = 1;
#pragma unroll
        for (int j = 0; j < SB; j++) row[j] = (j == CC) ? d : cmul(row[j], d);
        used = true;
        sm.prow[kglob & (HS_B - 1)] = pr;
        sm.perm[kglob] = pr;
        sm.pinv[pr] = kglob;
    } else {
        const cplx f = cmul(x, d);
#pragma unroll
        for (int j = 0; j < SB; j++) {
            const cplx pj = sm.crow[(pb + pw) * SB + j];
            if (j == CC) row[j] = cmake(-f.x, -f.y);
            else cfnma(row[j], f, pj);
        }
    }
}

// ---- panel factorisation in shared memory: columns [k0, k0 + bw) of all n rows --------------------
// On entry sm.panel[r][c] = X[r][k0 + c] (zero for c >= bw, r >= n).  On exit sm.panel = N' (the
// transformed columns), sm.prow[c] = pivot row of column k0 + c, perm / pinv updated, used |= pivot.
__device__ __forceinline__ void hs_factor_panel(HSmem &sm, int n, int k0, int bw, bool &used, int *status_slot)
{
    constexpr int B = HS_B, SB = HS_SB, NT = HS_NT, LDP = HS_LDP, LDR = HS_LDR;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
    const int r = tid;
    const bool has_row = r < n;
    const int naw = (n + 31) >> 5;              // warps that own rows: only they take part in the pivot search
    cplx *panel = sm.panel;
    cplx *Rs = sm.R[0];                       // [SB][LDR] snapshot of the sub-block's pivot rows
    for (int s = 0; s < B / SB; s++) {
        const int c0 = s * SB;
        const int ncols = bw - c0 < SB ? bw - c0 : SB;
        if (ncols <= 0) break;
        cplx row[SB];
        if (has_row) {
#pragma unroll
            for (int j = 0; j < SB; j++) row[j] = panel[r * LDP + c0 + j];
        } else {
#pragma unroll
            for (int j = 0; j < SB; j++) row[j] = cmake(0.0, 0.0);
        }
        if (warp < naw) {
            const int kg = k0 + c0;
            hs_pivot_step<0>(sm, row, used, r, lane, warp, naw, kg, status_slot);
            if (ncols > 1) hs_pivot_step<1>(sm, row, used, r, lane, warp, naw, kg + 1, status_slot);
            if (ncols > 2) hs_pivot_step<2>(sm, row, used, r, lane, warp, naw, kg + 2, status_slot);
            if (ncols > 3) hs_pivot_step<3>(sm, row, used, r, lane, warp, naw, kg + 3, status_slot);
            if (ncols > 4) hs_pivot_step<4>(sm, row, used, r, lane, warp, naw, kg + 4, status_slot);
            if (ncols > 5) hs_pivot_step<5>(sm, row, used, r, lane, warp, naw, kg + 5, status_slot);
            if (ncols > 6) hs_pivot_step<6>(sm, row, used, r, lane, warp, naw, kg + 6, status_slot);
            if (ncols > 7) hs_pivot_step<7>(sm, row, used, r, lane, warp, naw, kg + 7, status_slot);
        }
        __syncthreads();
        if (has_row) {
#pragma unroll
            for (int j = 0; j < SB; j++) panel[r * LDP + c0 + j] = row[j];
        }
        const int nbmax = (bw + 7) / 8;
        if (nbmax > 1) {
            for (int e = tid; e < SB * B; e += NT) {
                const int k = e / B, c = e % B;
                if (c < c0 || c >= c0 + SB) Rs[k * LDR + c] = (k < ncols) ? panel[sm.prow[c0 + k] * LDP + c] : cmake(0.0, 0.0);
            }
            __syncthreads();
            // other panel columns: panel[:, J] += (N'_s - E_s) (n x 8) * Rs (8 x |J|) on DMMA.
            // warp -> 32 rows (warp & 3), column blocks of parity (warp >> 2)
            const int rbase = (warp & 3) * 32;
            if (rbase < n) {
                int pk[2];
#pragma unroll
                for (int q = 0; q < 2; q++) pk[q] = (q * 4 + t < ncols) ? sm.prow[c0 + q * 4 + t] : -1;
                cplx a[2][4];
#pragma unroll
                for (int q = 0; q < 2; q++)
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        const int rr = rbase + i * 8 + g;
                        a[q][i] = panel[rr * LDP + c0 + q * 4 + t];
                        if (rr == pk[q]) a[q][i].x -= 1.0;
                    }
                int cnt = 0;
                for (int nb = 0; nb < nbmax; nb++) {
                    if (nb == s) continue;
                    if (((cnt++) & 1) != (warp >> 2)) continue;
                    double cre[4][2], cim[4][2];
                    cplx *Cw = panel + rbase * LDP + nb * 8;
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        const cplx v0 = Cw[(i * 8 + g) * LDP + 2 * t], v1 = Cw[(i * 8 + g) * LDP + 2 * t + 1];
                        cre[i][0] = v0.x; cim[i][0] = v0.y; cre[i][1] = v1.x; cim[i][1] = v1.y;
                    }
#pragma unroll
                    for (int q = 0; q < 2; q++) {
                        const cplx bb = Rs[(q * 4 + t) * LDR + nb * 8 + g];
#pragma unroll
                        for (int i = 0; i < 4; i++) zmma884(cre[i], cim[i], a[q][i].x, a[q][i].y, -a[q][i].y, bb.x, bb.y);
                    }
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        Cw[(i * 8 + g) * LDP + 2 * t] = cmake(cre[i][0], cim[i][0]);
                        Cw[(i * 8 + g) * LDP + 2 * t + 1] = cmake(cre[i][1], cim[i][1]);
                    }
                }
            }
            __syncthreads();
        }
    }
}

// ---- R = C[prow[0..bw)][col0 .. col0+32) -> shared memory (cp.async.cg: L2, never a stale L1 line) --------
__device__ __forceinline__ void hs_stage_R(HSmem &sm, int buf, const cplx *Cg, int ld, int col0, int ncols, int bw)
{
    cplx *R = sm.R[buf];
#pragma unroll
    for (int it = 0; it < (HS_B * HS_B) / HS_NT; it++) {
        const int e = threadIdx.x + it * HS_NT, k = e / HS_B, c = e % HS_B;
        const bool ok = k < bw && col0 + c < ncols;
        cp_async16(R + k * HS_LDR + c, ok ? Cg + (long long)sm.prow[k] * ld + col0 + c : Cg, ok ? 16 : 0);
    }
    cp_async_commit();
}

// ---- C[:, col0 .. col0+32) += Mult (n x 32, sm.panel) * R (32 x 32, sm.R[buf]), in place in L2 -------------
// warp w owns rows [16 w, 16 w + 16): 2 x 4 DMMA blocks of 8 x 8 complex.
__device__ __forceinline__ void hs_update_chunk(const HSmem &sm, int buf, cplx *Cg, int ld, int n, int col0, int ncols, int kmax)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
    const int wr = warp * 16;
    if (wr >= n) return;
    double cre[2][4][2], cim[2][4][2];
#pragma unroll
    for (int i = 0; i < 2; i++) {
        const int rr = wr + i * 8 + g;
        const cplx *src = Cg + (long long)rr * ld + col0 + 2 * t;
#pragma unroll
        for (int j = 0; j < 4; j++) {
#pragma unroll
            for (int q = 0; q < 2; q++) {
                cplx v = cmake(0.0, 0.0);
                if (rr < n && col0 + j * 8 + 2 * t + q < ncols) v = ldcg(src + j * 8 + q);
                cre[i][j][q] = v.x; cim[i][j][q] = v.y;
            }
        }
    }
    const cplx *cA = sm.panel + wr * HS_LDP;
    const cplx *cB = sm.R[buf];
#pragma unroll 2
    for (int kk = 0; kk < kmax; kk += 4) {
        cplx a[2], bb[4];
#pragma unroll
        for (int i = 0; i < 2; i++) a[i] = cA[(i * 8 + g) * HS_LDP + kk + t];
#pragma unroll
        for (int j = 0; j < 4; j++) bb[j] = cB[(kk + t) * HS_LDR + j * 8 + g];
#pragma unroll
        for (int i = 0; i < 2; i++) {
            const double nai = -a[i].y;
#pragma unroll
            for (int j = 0; j < 4; j++) zmma884(cre[i][j], cim[i][j], a[i].x, a[i].y, nai, bb[j].x, bb[j].y);
        }
    }
#pragma unroll
    for (int i = 0; i < 2; i++) {
        const int rr = wr + i * 8 + g;
        cplx *dst = Cg + (long long)rr * ld + col0 + 2 * t;
#pragma unroll
        for (int j = 0; j < 4; j++)
#pragma unroll
            for (int q = 0; q < 2; q++)
                if (rr < n && col0 + j * 8 + 2 * t + q < ncols) dst[j * 8 + q] = cmake(cre[i][j][q], cim[i][j][q]);
    }
}

// ---- [X | W] <- A^-1 [I | W] in place (X holds A on entry); fills sm.perm / sm.pinv ------------------------
__device__ __forceinline__ void hs_gauss_jordan(HSmem &sm, cplx *X, cplx *W, int ld, int n, int nc, int *status_slot, long long *prof)
{
    long long tc = prof ? clock64() : 0;
#define HS_TICK(slot) do { if (prof) { long long now_ = clock64(); if (threadIdx.x == 0) prof[slot] += now_ - tc; tc = now_; } } while (0)
    const int tid = threadIdx.x;
    bool used = !(tid < n);
    const int nchm = (n + HS_B - 1) / HS_B, ncha = (nc + HS_B - 1) / HS_B;
    for (int k0 = 0; k0 < n; k0 += HS_B) {
        const int bw = (n - k0 < HS_B) ? (n - k0) : HS_B;
        for (int e = tid; e < HS_NMAX * HS_B; e += HS_NT) {
            const int rr = e / HS_B, c = e % HS_B;
            const bool ok = rr < n && c < bw;
            cp_async16(sm.panel + rr * HS_LDP + c, ok ? X + (long long)rr * ld + k0 + c : X, ok ? 16 : 0);
        }
        cp_async_commit();
        cp_async_wait<0>();
        __syncthreads();
        HS_TICK(1);
        hs_factor_panel(sm, n, k0, bw, used, status_slot);
        HS_TICK(2);
        // N' -> X[:, K];  then the panel becomes Mult = N' - E (E[prow[c]][c] = 1)
        for (int e = tid; e < n * HS_B; e += HS_NT) {
            const int rr = e / HS_B, c = e % HS_B;
            if (c < bw) X[(long long)rr * ld + k0 + c] = sm.panel[rr * HS_LDP + c];
        }
        __syncthreads();
        if (tid < bw) sm.panel[sm.prow[tid] * HS_LDP + tid].x -= 1.0;
        // chunk list: matrix chunks except the panel's own, then the propagator chunks
        const int skip = k0 / HS_B, total = nchm - 1 + ncha;
        const int kmax = (bw + 3) & ~3;
        auto chunk = [&](int q, cplx *&base, int &col0, int &ncols) {
            if (q < nchm - 1) { const int j = q < skip ? q : q + 1; base = X; col0 = j * HS_B; ncols = n; }
            else { base = W; col0 = (q - (nchm - 1)) * HS_B; ncols = nc; }
        };
        cplx *base = nullptr; int col0 = 0, ncols = 0;
        if (total > 0) { chunk(0, base, col0, ncols); hs_stage_R(sm, 0, base, ld, col0, ncols, bw); }
        HS_TICK(3);
        for (int q = 0; q < total; q++) {
            cp_async_wait<0>();
            __syncthreads();
            if (q + 1 < total) { cplx *b2; int c2, n2; chunk(q + 1, b2, c2, n2); hs_stage_R(sm, (q + 1) & 1, b2, ld, c2, n2, bw); }
            chunk(q, base, col0, ncols);
            hs_update_chunk(sm, q & 1, base, ld, n, col0, ncols, kmax);
        }
        __syncthreads();
        HS_TICK(4);
    }
#undef HS_TICK
}

// ---- assembly of A (into Xn) and of W = C P_prev (into Wn) for half-step (i, kind) -------------------------
// g_prev[k][m] = Xp[perm_prev[k]][pinv_prev[m]], P_prev[k][:] = Wp[perm_prev[k]][:]; blocks of 32 output rows,
// the physical rows they need staged in the (idle) panel buffer so that every L2 read is a full row.
__device__ __forceinline__ void hs_assemble(HSmem &sm, const HSweepArgs &a, int bl, int i, int kind, bool first,
                                            const cplx *Xp, const cplx *Wp, cplx *Xn, cplx *Wn)
{
    const int tid = threadIdx.x, M = a.M, L = a.L, ld = a.ldn, nc = M / 2;
    const int bz = a.bz0 + bl, d = bz / a.n_E, e = bz % a.n_E;
    const double t2 = a.t * a.t, E = a.energies[e];
    const double *eps = a.onsite + ((long long)d * L + i) * M;
    const long long MM = (long long)M * M;
    const int par = kind == 0 ? ((i + 1) & 1) : (i & 1);
    const int n = half_count(M, par), nprev = kind == 0 ? n : half_count(M, 1 - par);
    const uint8_t *mk = a.bond + ((long long)d * (L + 1) + i) * M;        // m'_{i-1}
    const uint8_t *mr = a.bond + ((long long)d * (L + 1) + L) * M;        // m'_{L-1}
    const uint8_t *hp = a.hop + ((long long)d * L + i) * M;
    cplx *stage = sm.panel;                                                // [<= 36][HS_NMAX]
    if (first) {
        // half-step 0 (B_0): g_prev = surface Green's function of the left lead (slice -1, same atoms j), W = I
        const cplx *gl = a.gL + (long long)e * MM;
        for (int idx = tid; idx < n * n; idx += HS_NT) {
            const int r = idx / n, c = idx % n, jr = 2 * r + par, jc = 2 * c + par;
            cplx v = cmake(0.0, 0.0);
            if (r == c) v = cmake(E - eps[jr], a.eta);
            if (mk[jr] && mk[jc]) { const cplx g = gl[(long long)jr * M + jc]; v.x -= t2 * g.x; v.y -= t2 * g.y; }
            Xn[(long long)r * ld + c] = v;
        }
        for (int idx = tid; idx < n * nc; idx += HS_NT) {
            const int r = idx / nc, c = idx % nc;
            Wn[(long long)r * ld + c] = cmake(r == c ? 1.0 : 0.0, 0.0);
        }
        return;
    }
    const cplx *gr = a.gR + (long long)e * MM;
    const bool last = (kind == 1 && i == L - 1);
    // per-row tables of this half-step (the candidate buffers of the pivot search are idle here):
    //   kind B: ra[r] = m'[r];                       ca[c] = m'[c] ? physical column of g_prev[.][c] : -1
    //   kind F: ra/rb[r] = lower / upper B neighbour; ca/cb[c] = physical column of that neighbour, or -1
    HSTab &tb = *reinterpret_cast<HSTab *>(sm.crow);
    if (tid < n) {
        const int r = tid;
        tb.eps[r] = E - eps[2 * r + par];
        if (kind == 0) {
            const int m = mk[2 * r + par] ? 1 : 0;
            tb.ra[r] = (short)m; tb.rb[r] = -1;
            tb.ca[r] = (short)(m ? sm.pinv_prev[r] : -1); tb.cb[r] = -1;
        } else {
            const int s0 = half_nbr(r, par, 0, M, hp), s1 = half_nbr(r, par, 1, M, hp);
            tb.ra[r] = (short)s0; tb.rb[r] = (short)s1;
            tb.ca[r] = (short)(s0 >= 0 ? sm.pinv_prev[s0] : -1);
            tb.cb[r] = (short)(s1 >= 0 ? sm.pinv_prev[s1] : -1);
        }
    }
    __syncthreads();
    for (int r0 = 0; r0 < n; r0 += 32) {
        const int r1 = (r0 + 32 < n) ? r0 + 32 : n;
        int slo = r0, shi = r1 - 1;
        if (kind == 1) { if (par == 0) slo = r0 - 1; else shi = r1; }
        if (slo < 0) slo = 0;
        if (shi > nprev - 1) shi = nprev - 1;
        const int nst = shi - slo + 1;
        for (int idx = tid; idx < nst * ld; idx += HS_NT) {
            const int sl = idx / ld, c = idx - sl * ld;
            cp_async16(stage + sl * HS_NMAX + c, Xp + (long long)sm.perm_prev[slo + sl] * ld + c, 16);
        }
        cp_async_commit();
        cp_async_wait<0>();
        __syncthreads();
        for (int idx = tid; idx < (r1 - r0) * n; idx += HS_NT) {
            const int rl = idx / n, c = idx - rl * n, r = r0 + rl;
            cplx v = cmake(0.0, 0.0);
            if (r == c) v = cmake(tb.eps[r], a.eta);
            const int ca = tb.ca[c], cb = tb.cb[c];
            double sx = 0.0, sy = 0.0;
            if (kind == 0) {
                if (tb.ra[r] && ca >= 0) { const cplx g = stage[(r - slo) * HS_NMAX + ca]; sx = g.x; sy = g.y; }
            } else {
                const int ua = tb.ra[r], ub = tb.rb[r];
                if (ua >= 0) {
                    const cplx *sr = stage + (ua - slo) * HS_NMAX;
                    if (ca >= 0) { const cplx g = sr[ca]; sx += g.x; sy += g.y; }
                    if (cb >= 0) { const cplx g = sr[cb]; sx += g.x; sy += g.y; }
                }
                if (ub >= 0) {
                    const cplx *sr = stage + (ub - slo) * HS_NMAX;
                    if (ca >= 0) { const cplx g = sr[ca]; sx += g.x; sy += g.y; }
                    if (cb >= 0) { const cplx g = sr[cb]; sx += g.x; sy += g.y; }
                }
            }
            v.x -= t2 * sx; v.y -= t2 * sy;
            if (last) {
                const int jr = 2 * r + par, jc = 2 * c + par;
                if (mr[jr] && mr[jc]) { const cplx g = gr[(long long)jr * M + jc]; v.x -= t2 * g.x; v.y -= t2 * g.y; }
            }
            Xn[(long long)r * ld + c] = v;
        }
        __syncthreads();
    }
    // W = C P_prev: coalesced rows straight from L2, 4 independent elements per thread in flight
    const int nel = n * nc;
    for (int base = 0; base < nel; base += 4 * HS_NT) {
        cplx va[4], vb[4];
        int rr[4], cc[4];
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const int idx = base + k * HS_NT + tid;
            va[k] = cmake(0.0, 0.0); vb[k] = cmake(0.0, 0.0);
            rr[k] = -1;
            if (idx < nel) {
                const int r = idx / nc, c = idx - r * nc;
                rr[k] = r; cc[k] = c;
                if (kind == 0) {
                    if (tb.ra[r]) va[k] = ldcg(Wp + (long long)sm.perm_prev[r] * ld + c);
                } else {
                    const int ua = tb.ra[r], ub = tb.rb[r];
                    if (ua >= 0) va[k] = ldcg(Wp + (long long)sm.perm_prev[ua] * ld + c);
                    if (ub >= 0) vb[k] = ldcg(Wp + (long long)sm.perm_prev[ub] * ld + c);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < 4; k++)
            if (rr[k] >= 0) Wn[(long long)rr[k] * ld + cc[k]] = cmake(a.t * (va[k].x + vb[k].x), a.t * (va[k].y + vb[k].y));
    }
    __syncthreads();          // the tables alias the pivot-search buffers
}

// ---- the sweep: one CTA per matrix, half-steps [hs_begin, hs_end) ----------------------------------------
__global__ void __launch_bounds__(HS_NT, 2) half_sweep_kernel(HSweepArgs a)
{
    extern __shared__ __align__(16) unsigned char hs_smem_raw[];
    HSmem &sm = *reinterpret_cast<HSmem *>(hs_smem_raw);
    const int bl = blockIdx.x, tid = threadIdx.x, M = a.M, ld = a.ldn, nc = M / 2;
    const long long xs = (long long)ld * ld;
    cplx *Xb[2] = {a.X0 + bl * xs, a.X1 + bl * xs};
    cplx *Wb[2] = {a.P0 + bl * xs, a.P1 + bl * xs};
    int *gperm = a.perm + (long long)bl * HS_NMAX;
    int *status_slot = a.status + bl;
    if (a.hs_begin > 0) {
        if (tid < HS_NMAX) sm.perm[tid] = gperm[tid];
        __syncthreads();
        const int hp_ = a.hs_begin - 1, ip = hp_ >> 1, kp = hp_ & 1;
        const int np = half_count(M, kp == 0 ? ((ip + 1) & 1) : (ip & 1));
        if (tid < np) sm.pinv[sm.perm[tid]] = tid;
        __syncthreads();
    }
    int n = 0;
    for (int hs = a.hs_begin; hs < a.hs_end; hs++) {
        const int i = hs >> 1, kind = hs & 1, cur = hs & 1;
        if (tid < HS_NMAX) { sm.perm_prev[tid] = sm.perm[tid]; sm.pinv_prev[tid] = sm.pinv[tid]; }
        __syncthreads();
        long long tc0 = a.prof ? clock64() : 0;
        hs_assemble(sm, a, bl, i, kind, hs == 0, Xb[cur], Wb[cur], Xb[cur ^ 1], Wb[cur ^ 1]);
        __syncthreads();
        if (a.prof && tid == 0) a.prof[bl * 8 + 0] += clock64() - tc0;
        n = half_count(M, kind == 0 ? ((i + 1) & 1) : (i & 1));
        hs_gauss_jordan(sm, Xb[cur ^ 1], Wb[cur ^ 1], ld, n, nc, status_slot, a.prof ? a.prof + bl * 8 : nullptr);
    }
    if (tid < HS_NMAX) gperm[tid] = sm.perm[tid];
    if (a.hs_end > a.hs_begin && (a.g_out || a.P_out)) {
        const int fin = a.hs_end & 1;                  // buffer written by the last half-step
        const long long os = (long long)a.nh * a.nh;
        if (a.g_out)
            for (int idx = tid; idx < n * n; idx += HS_NT) {
                const int k = idx / n, m = idx % n;
                a.g_out[bl * os + idx] = ldcg(Xb[fin] + (long long)sm.perm[k] * ld + sm.pinv[m]);
            }
        if (a.P_out)
            for (int idx = tid; idx < n * nc; idx += HS_NT) {
                const int k = idx / nc, c = idx % nc;
                a.P_out[bl * os + (long long)k * a.nh + c] = ldcg(Wb[fin] + (long long)sm.perm[k] * ld + c);
            }
    }
}

}  // namespace rgf
