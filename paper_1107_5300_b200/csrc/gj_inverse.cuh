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
//   pivrow[B] cplx | red_val[32] double | red_idx[32] int | rowAt[n] int | posOf[n] int |
//   moved[2B] int | nmoved | stage[2B][GJ_CH] cplx
// ------------------------------------------------------------------------------------------
constexpr int GJ_CH = 32;   // columns per chunk when moving exchanged rows

template <int B>
__host__ __device__ constexpr size_t gj_panel_smem(int n)
{
    return sizeof(cplx) * B + sizeof(double) * 32 + sizeof(int) * 32 + sizeof(int) * 2 * (size_t)n +
           sizeof(int) * (2 * B + 4) + sizeof(cplx) * 2 * B * GJ_CH + 64;
}

template <int B, int NT, int ROWS>
__global__ void __launch_bounds__(NT) gj_panel_kernel(cplx *Gall, long long g_batch, int n, int k0,
                                                      cplx *Nall, cplx *Rall, int *origall, int *status)
{
    extern __shared__ __align__(16) unsigned char gj_smem[];
    cplx *pivrow = reinterpret_cast<cplx *>(gj_smem);
    double *red_val = reinterpret_cast<double *>(pivrow + B);
    int *red_idx = reinterpret_cast<int *>(red_val + 32);
    int *rowAt = red_idx + 32;
    int *posOf = rowAt + n;
    int *moved = posOf + n;
    int *nmoved = moved + 2 * B;
    cplx *stage = reinterpret_cast<cplx *>((reinterpret_cast<uintptr_t>(nmoved + 4) + 15) & ~(uintptr_t)15);

    const int b = blockIdx.x;
    cplx *G = Gall + (long long)b * g_batch;
    cplx *Nbuf = Nall + (long long)b * n * B;
    cplx *Rbuf = Rall + (long long)b * n * B;
    int *orig = origall + (long long)b * n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int bw = (n - k0 < B) ? (n - k0) : B;

    // thread tid owns rows tid, tid + NT, ... (ROWS of them), each with its B panel entries in registers
    cplx row[ROWS][B];
    bool used[ROWS];
#pragma unroll
    for (int q = 0; q < ROWS; q++) {
        const int r = tid + q * NT;
#pragma unroll
        for (int c = 0; c < B; c++) row[q][c] = (r < n && c < bw) ? G[(long long)r * n + k0 + c] : cmake(0.0, 0.0);
        used[q] = (r >= n || r < k0);     // positions < k0 hold the pivot rows of earlier panels
    }
    for (int i = tid; i < n; i += NT) { rowAt[i] = i; posOf[i] = i; }
    __syncthreads();

    // The column loop is a real loop (an unrolled one is ~400 KB of straight-line code and runs at
    // instruction-fetch speed); the register-resident row is indexed with select chains instead.
#pragma unroll 1
    for (int c = 0; c < bw; c++) {
        cplx x[ROWS];
        double v = -1.0;
        int idx = tid;
#pragma unroll
        for (int q = 0; q < ROWS; q++) {
            x[q] = row[q][0];
#pragma unroll
            for (int j = 1; j < B; j++) if (j == c) x[q] = row[q][j];
            // ---- pivot search: max |x|^2 over unused rows, lowest row index on ties
            double vq = used[q] ? -1.0 : cabs2(x[q]);
            if (!(vq == vq)) vq = 1e300;          // NaN: make it win so that it is reported
            if (vq > v) { v = vq; idx = tid + q * NT; }
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            double ov = __shfl_xor_sync(0xffffffffu, v, off);
            int oi = __shfl_xor_sync(0xffffffffu, idx, off);
            if (ov > v || (ov == v && oi < idx)) { v = ov; idx = oi; }
        }
        if (lane == 0) { red_val[warp] = v; red_idx[warp] = idx; }
        __syncthreads();
        double bv = red_val[0]; int pr = red_idx[0];
#pragma unroll
        for (int w = 1; w < NT / 32; w++) {
            double ov = red_val[w]; int oi = red_idx[w];
            if (ov > bv || (ov == bv && oi < pr)) { bv = ov; pr = oi; }
        }
#pragma unroll
        for (int q = 0; q < ROWS; q++) {
            if (tid + q * NT == pr) {
                if (!(bv > 0.0) || !(bv < 1e299)) status[b] = 1;          // zero / non-finite pivot
                cplx d = crecip(x[q]);
#pragma unroll
                for (int j = 0; j < B; j++) {
                    cplx y = (j == c) ? cmake(1.0, 0.0) : row[q][j];
                    row[q][j] = cmul(y, d);
                    pivrow[j] = row[q][j];
                }
                used[q] = true;
                // exchange positions k (= k0 + c) and the position currently holding row pr
                int k = k0 + c, a = rowAt[k], pp = posOf[pr];
                rowAt[k] = pr; posOf[pr] = k; rowAt[pp] = a; posOf[a] = pp;
            }
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < ROWS; q++) {
            if (tid + q * NT < n && tid + q * NT != pr) {
#pragma unroll
                for (int j = 0; j < B; j++) {
                    cplx y = (j == c) ? cmake(0.0, 0.0) : row[q][j];
                    cfnma(y, x[q], pivrow[j]);
                    row[q][j] = y;
                }
            }
        }
        // pivrow / red_* are rewritten only after the next column's first barrier
    }
    __syncthreads();

    // ---- list of positions whose row changed
    if (tid == 0) *nmoved = 0;
    __syncthreads();
    for (int i = tid; i < n; i += NT)
        if (rowAt[i] != i) { int q = atomicAdd(nmoved, 1); moved[q] = i; }
    __syncthreads();
    const int nm = *nmoved;                      // <= 2B

    // ---- new panel columns and multipliers (row r now lives at position posOf[r])
#pragma unroll
    for (int q = 0; q < ROWS; q++) {
        const int r = tid + q * NT;
        if (r < n) {
            const int pos = posOf[r];
#pragma unroll
            for (int c = 0; c < B; c++) {
                if (c < bw) G[(long long)pos * n + k0 + c] = row[q][c];
                cplx m = row[q][c];
                if (pos == k0 + c) m.x -= 1.0;
                Nbuf[(long long)pos * B + c] = (c < bw) ? m : cmake(0.0, 0.0);
            }
        }
    }
    // ---- origin bookkeeping: orig[pos] <- orig[rowAt[pos]]
    int my_orig = 0;
    if (tid < nm) my_orig = orig[rowAt[moved[tid]]];
    __syncthreads();
    if (tid < nm) orig[moved[tid]] = my_orig;

    // ---- move the exchanged rows in all non-panel columns, chunk by chunk
    for (int j0 = 0; j0 < n; j0 += GJ_CH) {
        for (int e = tid; e < nm * GJ_CH; e += NT) {
            int q = e / GJ_CH, j = j0 + e % GJ_CH;
            if (j < n && (j < k0 || j >= k0 + B)) stage[q * GJ_CH + (j - j0)] = G[(long long)rowAt[moved[q]] * n + j];
        }
        __syncthreads();
        for (int e = tid; e < nm * GJ_CH; e += NT) {
            int q = e / GJ_CH, j = j0 + e % GJ_CH;
            if (j < n && (j < k0 || j >= k0 + B)) G[(long long)moved[q] * n + j] = stage[q * GJ_CH + (j - j0)];
        }
        __syncthreads();
    }
    // ---- pivot rows (after the exchange, before the update) for the update kernel
    for (int e = tid; e < B * n; e += NT) {
        int c = e / n, j = e % n;
        Rbuf[(long long)c * n + j] = (c < bw) ? G[(long long)(k0 + c) * n + j] : cmake(0.0, 0.0);
    }
}

// ------------------------------------------------------------------------------------------
// Trailing update on the FP64 tensor pipe: G[:,J] += Nbuf (n x B) * Rbuf[:,J] (B x |J|).
// CTA = 4 warps stacked on rows: tile 128 rows x 32 columns; the Mult and pivot-row tiles are staged by TMA bulk copies
// (cp.async.bulk + mbarrier: BASELINE.json north_star "Large M uses TMA-staged panels"); the accumulators are initialised
// from G and stored back in place (each element is read and written by exactly one lane).
// 8-column blocks inside the panel [k0, k0+B) are skipped.
// ------------------------------------------------------------------------------------------
constexpr int GU_BM = 128, GU_BN = 32, GU_THREADS = 128;
template <int B> constexpr int gu_ldn() { return B + 4; }
constexpr int GU_LDR = GU_BN + 2;
template <int B> constexpr int gu_smem() { return (GU_BM * gu_ldn<B>() + B * GU_LDR) * (int)sizeof(cplx); }

template <int B>
__global__ void __launch_bounds__(GU_THREADS) gj_update_kernel(cplx *Gall, long long g_batch, int n, int k0,
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
    int nb_valid = (n - col0 + 7) / 8; nb_valid = nb_valid > 4 ? 4 : nb_valid;
    bool skipj[4];
#pragma unroll
    for (int j = 0; j < 4; j++) { int c = col0 + j * 8; skipj[j] = (j >= nb_valid) || (c >= k0 && c + 8 <= k0 + B); }

    double cre[4][4][2], cim[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) {
            int rr = wr + i * 8 + g, c = col0 + j * 8 + 2 * t;
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
        cplx a[4], bb[4];
#pragma unroll
        for (int i = 0; i < 4; i++) a[i] = cA[(i * 8 + g) * LDN + kk + t];
#pragma unroll
        for (int j = 0; j < 4; j++) bb[j] = sR[(kk + t) * GU_LDR + j * 8 + g];
#pragma unroll
        for (int i = 0; i < 4; i++)
            if (i < mb_valid) {
                double nai = -a[i].y;
#pragma unroll
                for (int j = 0; j < 4; j++)
                    if (!skipj[j]) zmma884(cre[i][j], cim[i][j], a[i].x, a[i].y, nai, bb[j].x, bb[j].y);
            }
    }
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) {
            int rr = wr + i * 8 + g, c = col0 + j * 8 + 2 * t;
            if (i < mb_valid && !skipj[j] && rr < n) {
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
