// gj_inverse32.cuh -- the fast path of the batched complex128 inverse for n <= 256 (the paper's
// 30 nm ribbon is n = 244): blocked Gauss-Jordan with partial pivoting, panels of 32 columns,
// ping-pong buffers X -> Y so that row exchanges cost nothing.
//
// One panel step k (columns K = [k0, k0+32)), for every matrix of the batch:
//   gj32_panel_kernel : reads X[:, K]; Gauss-Jordan with partial pivoting on the n x 32 panel held
//                       in shared memory, by hs_factor_panel of half_sweep.cuh (4 sub-blocks of 8 columns:
//                       pivot steps with the thread's row in registers, then one (n x 8) x (8 x 24) DMMA
//                       product for the other panel columns).  Rows are never moved; the
//                       exchange is the map rowAt[pos] = row of X that belongs at position pos.
//                       Writes Y[pos, K] = N'[rowAt[pos], :], Mult[pos, :] = N' - E, rowAt, orig.
//   gj32_update_kernel: Y[pos, J] = X[rowAt[pos], J] + Mult[pos, :] * X[rowAt[k0 + :], J]   (FP64 DMMA)
// then X <-> Y.  After the last panel gj32_unpermute_kernel scatters columns: out[:, orig[pos]] = X[:, pos].
// (Eq. 4 / PAPER.md:53 "one call of the linear equation solver".)
#pragma once
#include "half_sweep.cuh"
#include "rgf_common.cuh"

namespace rgf {

constexpr int G32_B = 32, G32_SB = 8, G32_NT = 256;
constexpr int G32_LDP = G32_B + 4;      // 36: A / C fragment accesses conflict-free
constexpr int G32_LDR = G32_B + 2;      // 34
__host__ __device__ constexpr size_t gj32_panel_smem(int n)
{
    return sizeof(cplx) * ((size_t)G32_NT * G32_LDP + G32_SB * G32_LDR + 2 * (G32_NT / 32) * (G32_SB + 1)) + sizeof(unsigned) * 4 * (G32_NT / 32) +
           sizeof(int) * (4 * (size_t)n + G32_B + 8) + 64;
}

// The factorisation itself is hs_factor_panel of half_sweep.cuh (one implementation of the pivot step and of the in-panel
// DMMA update for the fused kernel and for this one): thread = row, all eight warps search and update.
__global__ void __launch_bounds__(G32_NT) gj32_panel_kernel(const cplx *__restrict__ Xall, cplx *__restrict__ Yall, long long g_batch,
                                                            int n, int k0, cplx *__restrict__ Mall, int *__restrict__ rowAtAll,
                                                            int *__restrict__ origall, int *__restrict__ status)
{
    constexpr int B = G32_B, SB = G32_SB, NT = G32_NT, LDP = G32_LDP, LDR = G32_LDR;
    static_assert(G32_B == HS_B && G32_SB == HS_SB && G32_LDP == HS_LDP && G32_LDR == HS_LDR && G32_NT == HS_NT, "shares hs_factor_panel");
    extern __shared__ __align__(16) unsigned char gj_smem[];
    cplx *panel = reinterpret_cast<cplx *>(gj_smem);           // [NT][LDP], rows in X order
    cplx *Rs = panel + NT * LDP;                                // [SB][LDR] pivot rows of the sub-block
    cplx *crow = Rs + SB * LDR;                                 // [2][NT/32][SB] candidate pivot rows
    cplx *cinv = crow + 2 * (NT / 32) * SB;                     // [2][NT/32] 1 / candidate pivot
    unsigned *ckey = reinterpret_cast<unsigned *>(cinv + 2 * (NT / 32));               // [2][NT/32], 16-byte aligned
    unsigned *pivmin = ckey + 2 * (NT / 32);                                           // [1] (+ padding to 2 * NT / 32)
    int *rowAt = reinterpret_cast<int *>(pivmin + 2 * (NT / 32));
    int *posOf = rowAt + n;
    int *perm = posOf + n, *pinv = perm + n;                    // scratch of hs_factor_panel (pivot row of a column and back)
    int *prow = pinv + n;                                       // [B]

    const int b = blockIdx.x;
    const cplx *X = Xall + (long long)b * g_batch;
    cplx *Y = Yall + (long long)b * g_batch;
    cplx *Mult = Mall + (long long)b * n * B;
    int *orig = origall + (long long)b * n;
    int *rowAtG = rowAtAll + (long long)b * n;
    const int tid = threadIdx.x, warp = tid >> 5;
    const int r = tid;
    const bool has_row = r < n;
    const int bw = (n - k0 < B) ? (n - k0) : B;

    // ---- panel -> shared memory: one warp per row segment of 512 bytes, all copies in flight at once
    for (int e = tid; e < NT * B; e += NT) {
        int rr = e / B, c = e % B;
        bool ok = rr < n && c < bw;
        cp_async16(panel + rr * LDP + c, ok ? X + (long long)rr * n + k0 + c : X, ok ? 16 : 0);
    }
    cp_async_commit();
    for (int i = tid; i < n; i += NT) { rowAt[i] = i; posOf[i] = i; }
    bool used = (!has_row || r < k0);          // positions < k0 hold the pivot rows of earlier panels
    cp_async_wait<0>();
    __syncthreads();

    HSView v;
    v.panel = panel; v.Rs = Rs; v.crow = crow; v.cinv = cinv; v.ckey = ckey; v.prow = prow; v.perm = perm; v.pinv = pinv; v.pivmin = pivmin;
    HSGroup g;
    g.r = tid; g.slot = warp; g.nslots = (n + 31) >> 5; g.gtid = tid; g.gnt = NT;
    g.bar_pivot = 1; g.n_pivot = g.nslots * 32; g.bar_all = 0;
    g.rbase = warp * 32; g.nbsel = 0; g.nbmod = 1;
    hs_factor_panel<SB>(v, g, n, k0, bw, used, status + b);
    // the exchanges, in pivot order: position k0 + c takes row prow[c]
    if (tid == 0)
        for (int c = 0; c < bw; c++) {
            const int k = k0 + c, pr = prow[c], a = rowAt[k], pp = posOf[pr];
            rowAt[k] = pr; posOf[pr] = k; rowAt[pp] = a; posOf[a] = pp;
        }
    __syncthreads();

    // ---- outputs, in exchanged (position) order
    for (int e = tid; e < n * B; e += NT) {
        int pos = e / B, c = e % B;
        cplx v2 = panel[rowAt[pos] * LDP + c];
        if (c < bw) Y[(long long)pos * n + k0 + c] = v2;
        if (pos == k0 + c) v2.x -= 1.0;
        Mult[(long long)pos * B + c] = v2;
    }
    // orig[pos] <- orig[rowAt[pos]]; rowAt for the update kernel
    int o = 0;
    if (has_row) o = orig[rowAt[r]];
    __syncthreads();
    if (has_row) { orig[r] = o; rowAtG[r] = rowAt[r]; }
}

// ------------------------------------------------------------------------------------------
// Y[pos, J] = X[rowAt[pos], J] + Mult[pos, :] (n x 32) * X[rowAt[k0 + :], J] (32 x |J|), FP64 DMMA.
// CTA = 4 warps (2 x 2), 64 x 32 tile, warp tile 32 x 16: 53 KB of shared memory and ~110 registers, so
// that four CTAs share an SM and one CTA's loads / stores overlap the DMMAs of the others.
// 8-column blocks inside the panel are skipped.
// ------------------------------------------------------------------------------------------
constexpr int GU32_BM = 64, GU32_BN = 32, GU32_THREADS = 128, GU32_NB = GU32_BN / 16;
constexpr int GU32_LDN = G32_B + 4, GU32_LDR = GU32_BN + 2;
constexpr int GU32_SMEM = (GU32_BM * GU32_LDN + G32_B * GU32_LDR) * (int)sizeof(cplx);

__global__ void __launch_bounds__(GU32_THREADS, 4) gj32_update_kernel(const cplx *__restrict__ Xall, cplx *__restrict__ Yall, long long g_batch,
                                                                   int n, int k0, const cplx *__restrict__ Mall,
                                                                   const int *__restrict__ rowAtAll)
{
    constexpr int B = G32_B, LDN = GU32_LDN, LDR = GU32_LDR;
    extern __shared__ __align__(16) unsigned char gu_smem_raw[];
    cplx *sN = reinterpret_cast<cplx *>(gu_smem_raw);
    cplx *sR = sN + GU32_BM * LDN;

    const int b = blockIdx.z;
    const cplx *X = Xall + (long long)b * g_batch;
    cplx *Y = Yall + (long long)b * g_batch;
    const cplx *Mult = Mall + (long long)b * n * B;
    const int *rowAt = rowAtAll + (long long)b * n;
    const int row0 = blockIdx.y * GU32_BM, col0 = blockIdx.x * GU32_BN;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    // tile entirely inside the panel: nothing to do (a predicated-off DMMA still occupies the tensor pipe)
    if (col0 >= k0 && col0 + GU32_BN <= k0 + B) return;

    // the row maps this tile needs, fetched once (dependent global loads would otherwise serialise
    // every copy below behind a rowAt lookup)
    __shared__ int sRowK[G32_B], sRowM[GU32_BM];
    if (tid < G32_B) sRowK[tid] = (k0 + tid < n) ? rowAt[k0 + tid] : 0;
    else if (tid < G32_B + GU32_BM) { int rr = row0 + tid - G32_B; sRowM[tid - G32_B] = rr < n ? rowAt[rr] : 0; }
#pragma unroll
    for (int it = 0; it < (GU32_BM * B) / GU32_THREADS; it++) {
        int e = tid + it * GU32_THREADS, rr = e / B, k = e % B;
        bool ok = row0 + rr < n;
        cp_async16(sN + rr * LDN + k, ok ? Mult + (long long)(row0 + rr) * B + k : Mult, ok ? 16 : 0);
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < (B * GU32_BN) / GU32_THREADS; it++) {
        int e = tid + it * GU32_THREADS, k = e / GU32_BN, c = e % GU32_BN;
        bool ok = col0 + c < n && k0 + k < n;
        cp_async16(sR + k * LDR + c, ok ? X + (long long)sRowK[k] * n + col0 + c : X, ok ? 16 : 0);
    }
    cp_async_commit();

    constexpr int NB = GU32_NB;
    const int wr = row0 + (warp >> 1) * 32, wc = col0 + (warp & 1) * (8 * NB);
    int mb_valid = (n - wr + 7) / 8; mb_valid = mb_valid < 0 ? 0 : (mb_valid > 4 ? 4 : mb_valid);
    int nb_valid = (n - wc + 7) / 8; nb_valid = nb_valid < 0 ? 0 : (nb_valid > NB ? NB : nb_valid);
    bool skipj[NB];
#pragma unroll
    for (int j = 0; j < NB; j++) { int c = wc + j * 8; skipj[j] = (j >= nb_valid) || (c >= k0 && c < k0 + B); }

    double cre[4][NB][2], cim[4][NB][2];
#pragma unroll
    for (int i = 0; i < 4; i++) {
        const int rr = wr + i * 8 + g;
        const cplx *src = X + (long long)((i < mb_valid && rr < n) ? sRowM[rr - row0] : 0) * n;
#pragma unroll
        for (int j = 0; j < NB; j++) {
            const int c = wc + j * 8 + 2 * t;
#pragma unroll
            for (int q = 0; q < 2; q++) {
                cplx v = cmake(0.0, 0.0);
                if (i < mb_valid && !skipj[j] && rr < n && c + q < n) v = src[c + q];
                cre[i][j][q] = v.x; cim[i][j][q] = v.y;
            }
        }
    }
    cp_async_wait<0>();
    __syncthreads();
    const cplx *cA = sN + (warp >> 1) * 32 * LDN;
    const cplx *cB = sR + (warp & 1) * (8 * NB);
#pragma unroll
    for (int kk = 0; kk < B; kk += 4) {
        cplx a[4], bb[NB];
#pragma unroll
        for (int i = 0; i < 4; i++) a[i] = cA[(i * 8 + g) * LDN + kk + t];
#pragma unroll
        for (int j = 0; j < NB; j++) bb[j] = cB[(kk + t) * LDR + j * 8 + g];
#pragma unroll
        for (int i = 0; i < 4; i++)
            if (i < mb_valid) {
                const double nai = -a[i].y;
#pragma unroll
                for (int j = 0; j < NB; j++)
                    if (!skipj[j]) zmma884(cre[i][j], cim[i][j], a[i].x, a[i].y, nai, bb[j].x, bb[j].y);
            }
    }
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < NB; j++) {
            const int rr = wr + i * 8 + g, c = wc + j * 8 + 2 * t;
            if (i < mb_valid && !skipj[j] && rr < n) {
#pragma unroll
                for (int q = 0; q < 2; q++)
                    if (c + q < n) Y[(long long)rr * n + c + q] = cmake(cre[i][j][q], cim[i][j][q]);
            }
        }
}

// out[r][orig[pos]] = X[r][pos]: one warp per row, out of place
__global__ void gj32_unpermute_kernel(const cplx *__restrict__ Xall, cplx *__restrict__ Yall, long long g_batch, int n,
                                      const int *__restrict__ origall)
{
    const int b = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    const int r = blockIdx.x * nw + warp;
    if (r >= n) return;
    const cplx *src = Xall + (long long)b * g_batch + (long long)r * n;
    cplx *dst = Yall + (long long)b * g_batch + (long long)r * n;
    const int *orig = origall + (long long)b * n;
    for (int j = lane; j < n; j += 32) dst[orig[j]] = src[j];
}

}  // namespace rgf
