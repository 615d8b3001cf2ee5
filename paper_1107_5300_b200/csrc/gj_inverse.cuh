// gj_inverse.cuh -- batched complex128 inverse by blocked Gauss-Jordan with partial pivoting.
//
// G_ii = A_i^-1 is "one call of the linear equation solver" per recursion loop in the paper
// (Eq. 4).  Here it is an in-place blocked
// Gauss-Jordan elimination over panels of B columns, batched over (device, energy):
//
//   for each panel K = [k0, k0+B):
//     gj_panel_kernel  (one CTA per matrix, one thread per row, the row's B panel entries in
//                       registers): unblocked Gauss-Jordan with partial pivoting on the n x B
//                       panel; applies the row exchanges to the whole matrix; leaves
//                         G[:,K]  = N'        (transformed panel = columns K of the block transform)
//                         Nbuf    = N' - E_K  (n x B multipliers)
//                         Rbuf    = G[K,:]    (the B pivot rows before the update)
//     gj_update_kernel (FP64 tensor cores): G[:,J] += Nbuf * Rbuf[:,J] for all columns J not in K
//   gj_unpermute_kernel: A^-1[:, orig[pos]] = G[:, pos]  (undo the row exchanges as a column scatter)
//
// Why this shape: every panel step is the same n x (n-B) x B contraction (no shrinking trailing
// matrix), all O(n^3) work is DMMA, and the latency-bound pivot search of one matrix overlaps with
// the panels of the other matrices resident on the SM.
#pragma once
#include "rgf_common.cuh"
#include "zgemm.cuh"

namespace rgf {

// ------------------------------------------------------------------------------------------
// Panel factorisation.  blockDim.x = NT, NT * ROWS >= n (thread tid owns rows tid + q NT).  Dynamic shared memory:
//   crow[2][NT/32][B] cplx | cinv[2][NT/32] cplx | ckey[2][NT/32] unsigned | rowAt[n] int | posOf[n] int |
//   moved[2B] int | nmoved
// The pivot step is the fused kernel's (half_sweep.cuh, hs_pivot_step), widened to NT / 32 candidate warps and B columns:
// integer search key, every warp's candidate computes its own reciprocal before the one barrier of the step, the pivot row
// is not a divergent branch.
// ------------------------------------------------------------------------------------------
constexpr int GJ_XPER = 8;  // elements per thread and pass when moving exchanged rows

template <int B, int NT>
__host__ __device__ constexpr size_t gj_panel_smem(int n)
{
    return sizeof(cplx) * 2 * (NT / 32) * B + sizeof(cplx) * 2 * (NT / 32) + sizeof(unsigned) * 2 * (NT / 32) +
           sizeof(int) * 2 * (size_t)n + sizeof(int) * (2 * B + 4) + 64;
}

struct GJPanelSm {
    cplx *crow, *cinv;
    unsigned *ckey;
    int *rowAt, *posOf;
};

// One pivot step on column C (static) of the panel.  Key = top 21 bits of max(|re|, |im|) (exponent and 9 mantissa bits: a
// pivot within 2^-9 of the largest is as good as the largest) | (2047 - row): unique, names the row, lowest row wins ties.
// Candidate buffers alternate with the parity of C, so one barrier per column suffices.
//   row[j] <- c + a * pivrow[j]   with (a, c) = (d, 0) on the pivot row and (-x d, row[j]) elsewhere, row[C] <- a.
template <int C, int B, int NT, int ROWS>
__device__ __forceinline__ void gj_pivot_step(const GJPanelSm &sm, cplx (&row)[ROWS][B], bool (&used)[ROWS], int k0, int *status_b)
{
    constexpr int NW = NT / 32, pb = (C & 1) * NW;
    static_assert(NW % 4 == 0, "candidate keys are read four at a time");
    const int tid = threadIdx.x, warp = tid >> 5;
    unsigned key = 0u;
    int qs = 0;
#pragma unroll
    for (int q = 0; q < ROWS; q++) {
        const cplx x = row[q][C];
        const unsigned hre = (unsigned)__double2hiint(x.x) & 0x7fffffffu, him = (unsigned)__double2hiint(x.y) & 0x7fffffffu;
        const unsigned kq = (used[q] ? 0u : (max(hre, him) & 0xfffff800u)) | (unsigned)(2047 - (tid + q * NT));
        if (kq > key) { key = kq; qs = q; }
    }
    const unsigned wmax = __reduce_max_sync(0xffffffffu, key);
    if (key == wmax) {
#pragma unroll
        for (int q = 0; q < ROWS; q++)
            if (q == qs) {
                const cplx x = row[q][C];
                const double iv = hs_rcp(cabs2(x));
                sm.ckey[pb + warp] = key;
                sm.cinv[pb + warp] = cmake(x.x * iv, -x.y * iv);
#pragma unroll
                for (int j = 0; j < B; j++) if (j != C) sm.crow[(pb + warp) * B + j] = row[q][j];
            }
    }
    __syncthreads();
    unsigned best = 0u;
#pragma unroll
    for (int w = 0; w < NW; w += 4) {
        const uint4 k4 = *reinterpret_cast<const uint4 *>(&sm.ckey[pb + w]);
        best = max(max(best, max(k4.x, k4.y)), max(k4.z, k4.w));
    }
    const int pr = 2047 - (int)(best & 0x7ffu), pw = (pr % NT) >> 5;
    const cplx d = sm.cinv[pb + pw];
    const cplx *prow = sm.crow + (pb + pw) * B;
#pragma unroll
    for (int q = 0; q < ROWS; q++) {
        const cplx x = row[q][C];
        const bool is_piv = (tid + q * NT == pr);
        const cplx nf = cmake(fma(-x.x, d.x, x.y * d.y), fma(-x.x, d.y, -x.y * d.x));     // -(x d)
        const cplx a = is_piv ? d : nf;
#pragma unroll
        for (int j = 0; j < B; j++) {
            if (j == C) { row[q][j] = a; continue; }
            const cplx pj = prow[j];
            cplx c = is_piv ? cmake(0.0, 0.0) : row[q][j];
            c.x = fma(a.x, pj.x, c.x); c.x = fma(-a.y, pj.y, c.x);
            c.y = fma(a.x, pj.y, c.y); c.y = fma(a.y, pj.x, c.y);
            row[q][j] = c;
        }
        if (is_piv) {
            if ((best >> 11) == 0u || best >= 0x7ff00000u) *status_b = 1;          // zero / non-finite pivot
            used[q] = true;
            // exchange positions k (= k0 + C) and the position currently holding row pr
            const int k = k0 + C, ra = sm.rowAt[k], pp = sm.posOf[pr];
            sm.rowAt[k] = pr; sm.posOf[pr] = k; sm.rowAt[pp] = ra; sm.posOf[ra] = pp;
        }
    }
}

template <int C, int B, int NT, int ROWS>
__device__ __forceinline__ void gj_pivot_steps(const GJPanelSm &sm, cplx (&row)[ROWS][B], bool (&used)[ROWS], int k0, int bw, int *status_b)
{
    if constexpr (C < B) {
        if (C < bw) {
            gj_pivot_step<C, B, NT, ROWS>(sm, row, used, k0, status_b);
            gj_pivot_steps<C + 1, B, NT, ROWS>(sm, row, used, k0, bw, status_b);
        }
    }
}

template <int B, int NT, int ROWS>
__global__ void __launch_bounds__(NT) gj_panel_kernel(cplx *Gall, long long g_batch, int n, int k0,
                                                      cplx *Nall, cplx *Rall, int *origall, int *status)
{
    extern __shared__ __align__(16) unsigned char gj_smem[];
    constexpr int NW = NT / 32;
    GJPanelSm sm;
    sm.crow = reinterpret_cast<cplx *>(gj_smem);
    sm.cinv = sm.crow + 2 * NW * B;
    sm.ckey = reinterpret_cast<unsigned *>(sm.cinv + 2 * NW);
    sm.rowAt = reinterpret_cast<int *>(sm.ckey + 2 * NW);
    sm.posOf = sm.rowAt + n;
    int *rowAt = sm.rowAt, *posOf = sm.posOf;
    int *moved = posOf + n;
    int *nmoved = moved + 2 * B;

    const int b = blockIdx.x;
    cplx *G = Gall + (long long)b * g_batch;
    cplx *Nbuf = Nall + (long long)b * n * B;
    cplx *Rbuf = Rall + (long long)b * n * B;
    int *orig = origall + (long long)b * n;
    const int tid = threadIdx.x;
    const int bw = (n - k0 < B) ? (n - k0) : B;
    // 32-byte accesses to the panel columns of a row need (r n + k0) even for every r, and a full panel
    const bool vec = ((n & 1) == 0) && ((g_batch & 1) == 0) && bw == B && (reinterpret_cast<uintptr_t>(Gall) & 31) == 0;

    // thread tid owns rows tid, tid + NT, ... (ROWS of them), each with its B panel entries in registers
    cplx row[ROWS][B];
    bool used[ROWS];
#pragma unroll
    for (int q = 0; q < ROWS; q++) {
        const int r = tid + q * NT;
        if (vec && r < n) {
#pragma unroll
            for (int c = 0; c < B; c += 2)
                ld256cg(G + (long long)r * n + k0 + c, row[q][c].x, row[q][c].y, row[q][c + 1].x, row[q][c + 1].y);
        } else {
#pragma unroll
            for (int c = 0; c < B; c++) row[q][c] = (r < n && c < bw) ? G[(long long)r * n + k0 + c] : cmake(0.0, 0.0);
        }
        used[q] = (r >= n || r < k0);     // positions < k0 hold the pivot rows of earlier panels
    }
    for (int i = tid; i < n; i += NT) { rowAt[i] = i; posOf[i] = i; }
    if (tid < 2 * NW) sm.ckey[tid] = 0u;
    __syncthreads();

    gj_pivot_steps<0, B, NT, ROWS>(sm, row, used, k0, bw, status + b);
    __syncthreads();

    // ---- list of positions whose row changed
    if (tid == 0) *nmoved = 0;
    __syncthreads();
    for (int i = tid; i < n; i += NT)
        if (rowAt[i] != i) { int q = atomicAdd(nmoved, 1); moved[q] = i; }
    __syncthreads();
    const int nm = *nmoved;                      // <= 2B

    // ---- new panel columns and multipliers (row r now lives at position posOf[r]); 32-byte stores where aligned
#pragma unroll
    for (int q = 0; q < ROWS; q++) {
        const int r = tid + q * NT;
        if (r < n) {
            const int pos = posOf[r];
            if (vec) {
#pragma unroll
                for (int c = 0; c < B; c += 2)
                    st256(G + (long long)pos * n + k0 + c, row[q][c].x, row[q][c].y, row[q][c + 1].x, row[q][c + 1].y);
            } else {
#pragma unroll
                for (int c = 0; c < B; c++)
                    if (c < bw) G[(long long)pos * n + k0 + c] = row[q][c];
            }
#pragma unroll
            for (int c = 0; c < B; c += 2) {
                cplx m0 = row[q][c], m1 = row[q][c + 1];
                if (pos == k0 + c) m0.x -= 1.0;
                if (pos == k0 + c + 1) m1.x -= 1.0;
                if (c >= bw) m0 = cmake(0.0, 0.0);
                if (c + 1 >= bw) m1 = cmake(0.0, 0.0);
                st256(Nbuf + (long long)pos * B + c, m0.x, m0.y, m1.x, m1.y);
            }
        }
    }
    // ---- origin bookkeeping: orig[pos] <- orig[rowAt[pos]]
    int my_orig = 0;
    if (tid < nm) my_orig = orig[rowAt[moved[tid]]];
    __syncthreads();
    if (tid < nm) orig[moved[tid]] = my_orig;

    // ---- move the exchanged rows in all non-panel columns: passes over disjoint column ranges of cw columns (nm * cw <=
    // GJ_XPER * NT elements), every element of a pass loaded into registers before any is stored (one barrier per pass; passes
    // touch different columns, so nothing orders them against each other)
    if (nm > 0) {
        const int cw = (GJ_XPER * NT) / nm;
        for (int j0 = 0; j0 < n; j0 += cw) {
            const int wj = (n - j0 < cw) ? (n - j0) : cw, cnt = nm * wj;
            cplx v[GJ_XPER];
#pragma unroll
            for (int k = 0; k < GJ_XPER; k++) {
                const int e = k * NT + tid;
                if (e < cnt) {
                    const int q = e / wj, j = j0 + e - q * wj;
                    if (j < k0 || j >= k0 + B) v[k] = G[(long long)rowAt[moved[q]] * n + j];
                }
            }
            __syncthreads();
#pragma unroll
            for (int k = 0; k < GJ_XPER; k++) {
                const int e = k * NT + tid;
                if (e < cnt) {
                    const int q = e / wj, j = j0 + e - q * wj;
                    if (j < k0 || j >= k0 + B) G[(long long)moved[q] * n + j] = v[k];
                }
            }
        }
    }
    __syncthreads();
    // ---- pivot rows (after the exchange, before the update) for the update kernel
    for (int e0 = 0; e0 < B * n; e0 += GJ_XPER * NT) {          // GJ_XPER independent loads in flight per thread
        cplx v[GJ_XPER];
#pragma unroll
        for (int k = 0; k < GJ_XPER; k++) {
            const int e = e0 + k * NT + tid, c = e / n, j = e - c * n;
            v[k] = (e < B * n && c < bw) ? G[(long long)(k0 + c) * n + j] : cmake(0.0, 0.0);
        }
#pragma unroll
        for (int k = 0; k < GJ_XPER; k++) {
            const int e = e0 + k * NT + tid;
            if (e < B * n) Rbuf[e] = v[k];
        }
    }
}

// ------------------------------------------------------------------------------------------
// Trailing update on the FP64 tensor pipe: G[:,J] += Nbuf (n x B) * Rbuf[:,J] (B x |J|).
// CTA = 4 warps stacked on rows: tile 128 rows x 32 columns; the Mult and pivot-row tiles are staged by TMA bulk copies
// (cp.async.bulk + mbarrier: BASELINE.json north_star "Large M uses TMA-staged panels"); the accumulators are initialised
// from G and stored back in place (each element is read and written by exactly one lane).
// 8-column blocks inside the panel [k0, k0+B) are skipped.
// ------------------------------------------------------------------------------------------
constexpr int GU_BM = 128, GU_BN = 16, GU_THREADS = 128, GU_NJ = GU_BN / 8;
template <int B> constexpr int gu_ldn() { return B + 4; }
constexpr int GU_LDR = GU_BN + 2;
template <int B> constexpr int gu_smem() { return (GU_BM * gu_ldn<B>() + B * GU_LDR) * (int)sizeof(cplx); }

template <int B>
__global__ void __launch_bounds__(GU_THREADS, 4) gj_update_kernel(cplx *Gall, long long g_batch, int n, int k0,
                                                               const cplx *Nall, const cplx *Rall)
{
    extern __shared__ __align__(16) unsigned char gu_smem_raw[];
    cplx *sN = reinterpret_cast<cplx *>(gu_smem_raw);
    cplx *sR = sN + GU_BM * gu_ldn<B>();
    constexpr int LDN = gu_ldn<B>();

    const int b = blockIdx.z;
    cplx *G = Gall + (long long)b * g_batch;
    const cplx *Nbuf = Nall + (long long)b * n * B;
    const cplx *Rbuf = Rall + (long long)b * n * B;
    const int row0 = blockIdx.y * GU_BM, col0 = blockIdx.x * GU_BN;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    // whole tile inside the panel: nothing to do
    if (col0 >= k0 && col0 + GU_BN <= k0 + B) return;
    static_assert(B % 4 == 0, "panel width must be a multiple of the DMMA k");

    // stage Mult (rows row0 .., B columns: one contiguous row of the panel buffer each) and the B pivot rows (32 columns
    // from col0) with TMA bulk copies; rows / columns beyond n are not loaded (they only feed accumulators that are never stored)
    __shared__ unsigned long long bar;
    const int nrows = (n - row0 < GU_BM) ? (n - row0) : GU_BM, ncolsR = (n - col0 < GU_BN) ? (n - col0) : GU_BN;
    if (tid == 0) tma_bar_init(&bar, 1);
    __syncthreads();
    if (tid == 0) tma_expect(&bar, (unsigned)(nrows * B + B * ncolsR) * (unsigned)sizeof(cplx));
    for (int rr = tid; rr < nrows; rr += GU_THREADS)
        tma_load_row(sN + rr * LDN, Nbuf + (long long)(row0 + rr) * B, B * (unsigned)sizeof(cplx), &bar);
    for (int k = tid; k < B; k += GU_THREADS)
        tma_load_row(sR + k * GU_LDR, Rbuf + (long long)k * n + col0, ncolsR * (unsigned)sizeof(cplx), &bar);

    const int wr = row0 + warp * 32;
    int mb_valid = (n - wr + 7) / 8; mb_valid = mb_valid < 0 ? 0 : (mb_valid > 4 ? 4 : mb_valid);
    int nb_valid = (n - col0 + 7) / 8; nb_valid = nb_valid > GU_NJ ? GU_NJ : nb_valid;
    bool skipj[GU_NJ];
#pragma unroll
    for (int j = 0; j < GU_NJ; j++) { int c = col0 + j * 8; skipj[j] = (j >= nb_valid) || (c >= k0 && c + 8 <= k0 + B); }

    const bool vec = (B % 8 == 0) && ((n & 1) == 0) && ((g_batch & 1) == 0) && (reinterpret_cast<uintptr_t>(Gall) & 31) == 0;
    double cre[4][GU_NJ][2], cim[4][GU_NJ][2];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < GU_NJ; j++) {
            int rr = wr + i * 8 + g, c = col0 + j * 8 + 2 * t;
            if (vec) {
                // both elements of the lane in one 32-byte access (n even: c < n implies c + 1 < n; B % 8 == 0: a column block is inside
                // the panel or outside it as a whole)
                cre[i][j][0] = cim[i][j][0] = cre[i][j][1] = cim[i][j][1] = 0.0;
                if (i < mb_valid && !skipj[j] && rr < n && c < n)
                    ld256cg(G + (long long)rr * n + c, cre[i][j][0], cim[i][j][0], cre[i][j][1], cim[i][j][1]);
                continue;
            }
#pragma unroll
            for (int q = 0; q < 2; q++) {
                cplx v = cmake(0.0, 0.0);
                if (i < mb_valid && !skipj[j] && rr < n && c + q < n) v = G[(long long)rr * n + c + q];
                cre[i][j][q] = v.x; cim[i][j][q] = v.y;
            }
        }
    tma_wait(&bar, 0);
    const cplx *cA = sN + warp * 32 * LDN;
#pragma unroll
    for (int kk = 0; kk < B; kk += 4) {
        cplx a[4], bb[GU_NJ];
#pragma unroll
        for (int i = 0; i < 4; i++) a[i] = cA[(i * 8 + g) * LDN + kk + t];
#pragma unroll
        for (int j = 0; j < GU_NJ; j++) bb[j] = sR[(kk + t) * GU_LDR + j * 8 + g];
#pragma unroll
        for (int i = 0; i < 4; i++)
            if (i < mb_valid) {
                double nai = -a[i].y;
#pragma unroll
                for (int j = 0; j < GU_NJ; j++)
                    if (!skipj[j]) zmma884(cre[i][j], cim[i][j], a[i].x, a[i].y, nai, bb[j].x, bb[j].y);
            }
    }
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < GU_NJ; j++) {
            int rr = wr + i * 8 + g, c = col0 + j * 8 + 2 * t;
            if (i < mb_valid && !skipj[j] && rr < n) {
                if (vec) { if (c < n) st256(G + (long long)rr * n + c, cre[i][j][0], cim[i][j][0], cre[i][j][1], cim[i][j][1]); continue; }
#pragma unroll
                for (int q = 0; q < 2; q++)
                    if (c + q < n && !(c + q >= k0 && c + q < k0 + B))      // panel columns hold N' already
                        G[(long long)rr * n + c + q] = cmake(cre[i][j][q], cim[i][j][q]);
            }
        }
}

// A^-1[r][orig[pos]] = G[r][pos], in place row by row (one warp per row, row staged in shared memory).
__global__ void gj_unpermute_kernel(cplx *Gall, long long g_batch, int n, const int *origall)
{
    extern __shared__ __align__(16) unsigned char gp_smem[];
    cplx *buf = reinterpret_cast<cplx *>(gp_smem);
    const int b = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    const int r = blockIdx.x * nw + warp;
    if (r >= n) return;
    cplx *Grow = Gall + (long long)b * g_batch + (long long)r * n;
    const int *orig = origall + (long long)b * n;
    cplx *mybuf = buf + (size_t)warp * n;
    for (int j = lane; j < n; j += 32) mybuf[j] = Grow[j];
    __syncwarp();
    for (int j = lane; j < n; j += 32) Grow[orig[j]] = mybuf[j];
}

__global__ void gj_init_orig_kernel(int *origall, int n, int total)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < total) origall[i] = i % n;
}

}  // namespace rgf
