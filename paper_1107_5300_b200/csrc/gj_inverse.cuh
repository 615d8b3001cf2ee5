// gj_inverse.cuh -- batched complex128 inverse by blocked Gauss-Jordan with partial pivoting.
//
// G_ii = A_i^-1 is "one call of the linear equation solver" per recursion loop in the paper
// (Eq. 4).  Here it is an in-place blocked
// Gauss-Jordan elimination over panels of B columns, batched over (device, energy):
//
//   for each panel K = [k0, k0+B), ping-pong X -> Y as in gj_inverse32.cuh (rows are never moved):
//     gj_panel_kernel  (one CTA per matrix, one thread per row of X, the row's B panel entries in
//                       registers): unblocked Gauss-Jordan with partial pivoting on the n x B
//                       panel; the exchange is the map rowAt[pos] = row of X that belongs at position pos; leaves
//                         Y[pos,K]   = N'[rowAt[pos],:]  (transformed panel = columns K of the block transform)
//                         Nbuf[pos,:] = N' - E_K          (n x B multipliers)
//                         rowAt, orig
//     gj_update_kernel (FP64 tensor cores): Y[pos,J] = X[rowAt[pos],J] + Nbuf[pos,:] * X[rowAt[k0 + :],J] for all columns J not in K
//   then X <-> Y;  gj_unpermute_kernel: A^-1[:, orig[pos]] = X[:, pos]  (undo the exchanges as a column scatter)
//
// Why this shape: every panel step is the same n x (n-B) x B contraction (no shrinking trailing
// matrix), all O(n^3) work is DMMA, and the latency-bound pivot search of one matrix overlaps with
// the panels of the other matrices resident on the SM.  Round 2: the panel kernel used to exchange the rows physically and
// to snapshot the pivot rows for the update kernel -- 0.9 MB of traffic per 16-column panel through ONE SM per matrix, at
// the ~40 GB/s a single SM sustains against DRAM latency; with the ping-pong the update kernel's 2048 CTAs do the gather.
#pragma once
#include "rgf_common.cuh"
#include "zgemm.cuh"

namespace rgf {

// ------------------------------------------------------------------------------------------
// Panel factorisation.  blockDim.x = NT, NT * ROWS >= n (thread tid owns rows tid + q NT).  Dynamic shared memory:
//   crow[2][NT/32][B] cplx | cinv[2][NT/32] cplx | ckey[2][NT/32] unsigned | rowAt[n] int | posOf[n] int |
//   tr[NT/32][32 (B+1) + 8] cplx (per-warp transposition buffer of the epilogue + 32 positions)
// The pivot step is the fused kernel's (half_sweep.cuh, hs_pivot_step), widened to NT / 32 candidate warps and B columns:
// integer search key, every warp's candidate computes its own reciprocal before the one barrier of the step, the pivot row
// is not a divergent branch.
// ------------------------------------------------------------------------------------------
template <int B, int NT>
__host__ __device__ constexpr size_t gj_panel_smem(int n)
{
    return sizeof(cplx) * 2 * (NT / 32) * B + sizeof(cplx) * 2 * (NT / 32) + sizeof(unsigned) * 2 * (NT / 32) +
           sizeof(int) * 2 * (size_t)n + 64 + sizeof(cplx) * (NT / 32) * (32 * (B + 1) + 8);
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
__global__ void __launch_bounds__(NT) gj_panel_kernel(const cplx *Xall, cplx *Yall, long long g_batch, int n, int k0,
                                                      cplx *Nall, int *rowAtAll, int *origall, int *status)
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
    cplx *tr = reinterpret_cast<cplx *>((reinterpret_cast<uintptr_t>(posOf + n) + 15) & ~(uintptr_t)15);

    const int b = blockIdx.x;
    const cplx *X = Xall + (long long)b * g_batch;
    cplx *Y = Yall + (long long)b * g_batch;
    cplx *Nbuf = Nall + (long long)b * n * B;
    int *orig = origall + (long long)b * n;
    int *rowAtG = rowAtAll + (long long)b * n;
    const int tid = threadIdx.x;
    const int bw = (n - k0 < B) ? (n - k0) : B;
    // 32-byte accesses to the panel columns of a row need (r n + k0) even for every r, and a full panel
    const bool vec = ((n & 1) == 0) && ((g_batch & 1) == 0) && bw == B && ((reinterpret_cast<uintptr_t>(Xall) | reinterpret_cast<uintptr_t>(Yall)) & 31) == 0;

    // thread tid owns rows tid, tid + NT, ... (ROWS of them), each with its B panel entries in registers
    cplx row[ROWS][B];
    bool used[ROWS];
#pragma unroll
    for (int q = 0; q < ROWS; q++) {
        const int r = tid + q * NT;
        if (vec && r < n) {
#pragma unroll
            for (int c = 0; c < B; c += 2)
                ld256cg(X + (long long)r * n + k0 + c, row[q][c].x, row[q][c].y, row[q][c + 1].x, row[q][c + 1].y);
        } else {
#pragma unroll
            for (int c = 0; c < B; c++) row[q][c] = (r < n && c < bw) ? X[(long long)r * n + k0 + c] : cmake(0.0, 0.0);
        }
        used[q] = (r >= n || r < k0);     // positions < k0 hold the pivot rows of earlier panels
    }
    for (int i = tid; i < n; i += NT) { rowAt[i] = i; posOf[i] = i; }
    if (tid < 2 * NW) sm.ckey[tid] = 0u;
    __syncthreads();

    gj_pivot_steps<0, B, NT, ROWS>(sm, row, used, k0, bw, status + b);
    __syncthreads();

    // ---- new panel columns and multipliers (row r now lives at position posOf[r]).  Full panel, aligned rows: every warp
    // transposes its 32 rows through shared memory so that a store instruction writes whole 32-byte sectors of 64 / B rows
    // (B / 2 lanes per row) instead of one sector in each of 32 rows.
#pragma unroll
    for (int q = 0; q < ROWS; q++) {
        const int r = tid + q * NT;
        if (vec) {
            cplx *tw = tr + (size_t)(tid >> 5) * (32 * (B + 1) + 8);
            int *pw = reinterpret_cast<int *>(tw + 32 * (B + 1));
            const int lane = tid & 31;
#pragma unroll
            for (int c = 0; c < B; c++) tw[lane * (B + 1) + c] = row[q][c];
            pw[lane] = r < n ? posOf[r] : -1;
            __syncwarp();
            constexpr int LPR = B / 2, RPI = 32 / LPR;          // lanes per row, rows per instruction
#pragma unroll
            for (int it = 0; it < 32 / RPI; it++) {
                const int rr = it * RPI + lane / LPR, c = 2 * (lane % LPR), pos = pw[rr];
                if (pos >= 0) {
                    cplx m0 = tw[rr * (B + 1) + c], m1 = tw[rr * (B + 1) + c + 1];
                    st256(Y + (long long)pos * n + k0 + c, m0.x, m0.y, m1.x, m1.y);
                    if (pos == k0 + c) m0.x -= 1.0;
                    if (pos == k0 + c + 1) m1.x -= 1.0;
                    st256(Nbuf + (long long)pos * B + c, m0.x, m0.y, m1.x, m1.y);
                }
            }
            __syncwarp();
        } else if (r < n) {
            const int pos = posOf[r];
#pragma unroll
            for (int c = 0; c < B; c++) {
                if (c < bw) Y[(long long)pos * n + k0 + c] = row[q][c];
                cplx m = row[q][c];
                if (pos == k0 + c) m.x -= 1.0;
                Nbuf[(long long)pos * B + c] = (c < bw) ? m : cmake(0.0, 0.0);
            }
        }
    }
    // ---- origin bookkeeping orig[pos] <- orig[rowAt[pos]], and the map for the update kernel
    int o[ROWS];
#pragma unroll
    for (int q = 0; q < ROWS; q++) { const int r = tid + q * NT; o[q] = r < n ? orig[rowAt[r]] : 0; }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < ROWS; q++) { const int r = tid + q * NT; if (r < n) { orig[r] = o[q]; rowAtG[r] = rowAt[r]; } }
}

// ------------------------------------------------------------------------------------------
// Trailing update on the FP64 tensor pipe: Y[pos,J] = X[rowAt[pos],J] + Nbuf[pos,:] (n x B) * X[rowAt[k0 + :],J] (B x |J|).
// CTA = 4 warps stacked on rows: tile 128 rows x 16 columns (rank-16 updates are bound by HBM, not by the tensor pipe: a
// narrow tile keeps the accumulators at 64 registers so that four CTAs share an SM and their loads overlap); the Mult and
// pivot-row tiles are staged by TMA bulk copies (cp.async.bulk + mbarrier: BASELINE.json north_star "Large M uses
// TMA-staged panels"), the pivot rows straight from X through the row map; the accumulators are initialised from X and
// stored to Y with 32-byte accesses.  8-column blocks inside the panel [k0, k0+B) are skipped.
// ------------------------------------------------------------------------------------------
constexpr int GU_BM = 128, GU_BN = 16, GU_THREADS = 128, GU_NJ = GU_BN / 8;
template <int B> constexpr int gu_ldn() { return B + 4; }
constexpr int GU_LDR = GU_BN + 2;
template <int B> constexpr int gu_smem() { return (GU_BM * gu_ldn<B>() + B * GU_LDR) * (int)sizeof(cplx); }

template <int B>
__global__ void __launch_bounds__(GU_THREADS, 4) gj_update_kernel(const cplx *Xall, cplx *Yall, long long g_batch, int n, int k0,
                                                               const cplx *Nall, const int *rowAtAll)
{
    extern __shared__ __align__(16) unsigned char gu_smem_raw[];
    cplx *sN = reinterpret_cast<cplx *>(gu_smem_raw);
    cplx *sR = sN + GU_BM * gu_ldn<B>();
    constexpr int LDN = gu_ldn<B>();

    const int b = blockIdx.z;
    const cplx *X = Xall + (long long)b * g_batch;
    cplx *Y = Yall + (long long)b * g_batch;
    const cplx *Nbuf = Nall + (long long)b * n * B;
    const int *rowAt = rowAtAll + (long long)b * n;
    const int row0 = blockIdx.y * GU_BM, col0 = blockIdx.x * GU_BN;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    // whole tile inside the panel: nothing to do
    if (col0 >= k0 && col0 + GU_BN <= k0 + B) return;
    static_assert(B % 4 == 0, "panel width must be a multiple of the DMMA k");

    // stage Mult (rows row0 .., B columns: one contiguous row of the panel buffer each) and the B pivot rows (32 columns
    // from col0) with TMA bulk copies; rows / columns beyond n are not loaded (they only feed accumulators that are never stored)
    __shared__ unsigned long long bar;
    __shared__ int sRowM[GU_BM], sRowK[B];          // rows of X that belong at positions row0 .. row0 + 127 and k0 .. k0 + B - 1
    const int nrows = (n - row0 < GU_BM) ? (n - row0) : GU_BM, ncolsR = (n - col0 < GU_BN) ? (n - col0) : GU_BN;
    const int bw = (n - k0 < B) ? (n - k0) : B;
    if (tid == 0) tma_bar_init(&bar, 1);
    for (int rr = tid; rr < GU_BM; rr += GU_THREADS) sRowM[rr] = rr < nrows ? rowAt[row0 + rr] : 0;
    if (tid >= GU_THREADS - B) { const int k = tid - (GU_THREADS - B); sRowK[k] = k < bw ? rowAt[k0 + k] : 0; }
    // pivot rows beyond a narrow last panel: zero (their Mult columns are zero, but shared memory may hold NaN patterns)
    for (int e = tid; e < (B - bw) * GU_BN; e += GU_THREADS) sR[(bw + e / GU_BN) * GU_LDR + e % GU_BN] = cmake(0.0, 0.0);
    __syncthreads();
    if (tid == 0) tma_expect(&bar, (unsigned)(nrows * B + bw * ncolsR) * (unsigned)sizeof(cplx));
    for (int rr = tid; rr < nrows; rr += GU_THREADS)
        tma_load_row(sN + rr * LDN, Nbuf + (long long)(row0 + rr) * B, B * (unsigned)sizeof(cplx), &bar);
    for (int k = tid; k < bw; k += GU_THREADS)
        tma_load_row(sR + k * GU_LDR, X + (long long)sRowK[k] * n + col0, ncolsR * (unsigned)sizeof(cplx), &bar);

    const int wr = row0 + warp * 32;
    int mb_valid = (n - wr + 7) / 8; mb_valid = mb_valid < 0 ? 0 : (mb_valid > 4 ? 4 : mb_valid);
    int nb_valid = (n - col0 + 7) / 8; nb_valid = nb_valid > GU_NJ ? GU_NJ : nb_valid;
    bool skipj[GU_NJ];
#pragma unroll
    for (int j = 0; j < GU_NJ; j++) { int c = col0 + j * 8; skipj[j] = (j >= nb_valid) || (c >= k0 && c + 8 <= k0 + B); }

    const bool vec = (B % 8 == 0) && ((n & 1) == 0) && ((g_batch & 1) == 0) && ((reinterpret_cast<uintptr_t>(Xall) | reinterpret_cast<uintptr_t>(Yall)) & 31) == 0;
    double cre[4][GU_NJ][2], cim[4][GU_NJ][2];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < GU_NJ; j++) {
            int rr = wr + i * 8 + g, c = col0 + j * 8 + 2 * t;
            const cplx *src = X + (long long)((i < mb_valid && rr < n) ? sRowM[rr - row0] : 0) * n;
            if (vec) {
                // both elements of the lane in one 32-byte access (n even: c < n implies c + 1 < n; B % 8 == 0: a column block is inside
                // the panel or outside it as a whole)
                cre[i][j][0] = cim[i][j][0] = cre[i][j][1] = cim[i][j][1] = 0.0;
                if (i < mb_valid && !skipj[j] && rr < n && c < n)
                    ld256cg(src + c, cre[i][j][0], cim[i][j][0], cre[i][j][1], cim[i][j][1]);
                continue;
            }
#pragma unroll
            for (int q = 0; q < 2; q++) {
                cplx v = cmake(0.0, 0.0);
                if (i < mb_valid && !skipj[j] && rr < n && c + q < n) v = src[c + q];
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
                if (vec) { if (c < n) st256(Y + (long long)rr * n + c, cre[i][j][0], cim[i][j][0], cre[i][j][1], cim[i][j][1]); continue; }
#pragma unroll
                for (int q = 0; q < 2; q++)
                    if (c + q < n && !(c + q >= k0 && c + q < k0 + B))      // panel columns hold N' already
                        Y[(long long)rr * n + c + q] = cmake(cre[i][j][q], cim[i][j][q]);
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
