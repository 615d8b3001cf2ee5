// zgemm.cuh -- batched complex128 GEMM on the FP64 tensor pipe (DMMA.8x8x4) for sm_100a.
//
//   C[b] (Mr x Nc) = alpha * opA[b] (Mr x K) * B[b] (K x Nc)
//
// opA is addressed with arbitrary element strides (a_rs per row, a_cs per k), which covers
// plain, transposed and parity-gathered operands (the armchair propagator reads rows S_i and
// columns S_{i-1} of G_ii: stride 2 in both directions), optionally conjugated, optionally
// with whole k-columns zeroed by a byte mask (vacancy-aware bond mask).  B and C are row-major.
// Used by: the propagator G_{i,0} = G_ii V G_{i-1,0} (Eq. 5),
// the Sancho-Rubio products (A2) and the two contractions of the Gamma trace (A6).
//
// Tiling: CTA = 4 warps, 64 x 64 output tile, warp tile 32 x 32 = 4 x 4 DMMA blocks, BK = 16
// per stage, cp.async double buffering (one complex128 element = one 16-byte LDGSTS).
// Shared-memory leading dimensions are chosen so that the LDS.128 fragment loads are
// conflict-free: ldA = 4 (mod 8), ldB = 2 (mod 8) elements.
#pragma once
#include "rgf_common.cuh"

namespace rgf {

struct ZgemmArgs {
    const cplx *A; long long a_batch; long long a_rs, a_cs; int a_mod; int conjA;
    const uint8_t *kmask; long long kmask_batch; int kmask_div; int kmask_b0;   // optional: A(:,k) = 0 where kmask[k] == 0; mask row = (b0 + bz) / div
    const cplx *B; long long b_batch; int ldb; int b_mod;
    cplx *C; long long c_batch; int ldc;
    int Mr, Nc, K;
    cplx alpha;
};

constexpr int ZG_BM = 64, ZG_BN = 64, ZG_BK = 16, ZG_THREADS = 128;
constexpr int ZG_LDA = ZG_BK + 4;    // 20
constexpr int ZG_LDB = ZG_BN + 2;    // 66
constexpr int ZG_STAGES = 2;
constexpr int ZG_KMASK_MAX = 1024;     // masked GEMMs have K <= ceil(M/2) <= 512
constexpr int ZG_SMEM = ZG_STAGES * (ZG_BM * ZG_LDA + ZG_BK * ZG_LDB) * (int)sizeof(cplx);

// One k4 step of a warp tile of MB x NB DMMA blocks.  sA points at the warp's first row,
// sB at the warp's first column; kk is the k offset inside the staged chunk.
template <int MB, int NB>
__device__ __forceinline__ void warp_zmma_k4(double (&cre)[MB][NB][2], double (&cim)[MB][NB][2],
                                             const cplx *sA, int ldA, const cplx *sB, int ldB, int kk,
                                             int mb_valid, int nb_valid, int g, int t, double asign = 1.0)
{
    cplx a[MB], b[NB];
#pragma unroll
    for (int i = 0; i < MB; i++) { a[i] = sA[(i * 8 + g) * ldA + kk + t]; a[i].y *= asign; }
#pragma unroll
    for (int j = 0; j < NB; j++) b[j] = sB[(kk + t) * ldB + j * 8 + g];
#pragma unroll
    for (int i = 0; i < MB; i++) {
        if (i < mb_valid) {
            double nai = -a[i].y;
#pragma unroll
            for (int j = 0; j < NB; j++)
                if (j < nb_valid) zmma884(cre[i][j], cim[i][j], a[i].x, a[i].y, nai, b[j].x, b[j].y);
        }
    }
}

__global__ void __launch_bounds__(ZG_THREADS) zgemm_kernel(ZgemmArgs p)
{
    extern __shared__ __align__(16) unsigned char zg_smem[];
    cplx *sA = reinterpret_cast<cplx *>(zg_smem);
    cplx *sB = sA + ZG_STAGES * ZG_BM * ZG_LDA;

    const int bz = blockIdx.z;
    const cplx *A = p.A + (long long)(p.a_mod > 0 ? bz % p.a_mod : bz) * p.a_batch;
    const cplx *B = p.B + (long long)(p.b_mod > 0 ? bz % p.b_mod : bz) * p.b_batch;
    cplx *C = p.C + (long long)bz * p.c_batch;
    const uint8_t *kmask = p.kmask ? p.kmask + (long long)((p.kmask_b0 + bz) / p.kmask_div) * p.kmask_batch : nullptr;
    const int row0 = blockIdx.y * ZG_BM, col0 = blockIdx.x * ZG_BN;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, g = lane >> 2, t = lane & 3;
    const int wr = (warp >> 1) * 32, wc = (warp & 1) * 32;
    const bool k_fast = p.a_cs <= p.a_rs;
    // k mask staged once: a global byte load in front of every copy would serialise the stage loads
    __shared__ uint8_t sKmask[ZG_KMASK_MAX];
    const bool masked = kmask != nullptr;
    if (masked) {
        for (int k = tid; k < p.K && k < ZG_KMASK_MAX; k += ZG_THREADS) sKmask[k] = kmask[k];
        __syncthreads();
    }

    auto load_stage = [&](int stage, int k0) {
        cplx *dA = sA + stage * ZG_BM * ZG_LDA;
        cplx *dB = sB + stage * ZG_BK * ZG_LDB;
#pragma unroll
        for (int e = 0; e < (ZG_BM * ZG_BK) / ZG_THREADS; e++) {
            int idx = tid + e * ZG_THREADS, r, k;
            if (k_fast) { r = idx / ZG_BK; k = idx % ZG_BK; } else { k = idx / ZG_BM; r = idx % ZG_BM; }
            int gr = row0 + r, gk = k0 + k;
            bool ok = gr < p.Mr && gk < p.K && (!masked || sKmask[gk]);
            const cplx *src = ok ? A + (long long)gr * p.a_rs + (long long)gk * p.a_cs : A;
            cp_async16(dA + r * ZG_LDA + k, src, ok ? 16 : 0);
        }
#pragma unroll
        for (int e = 0; e < (ZG_BK * ZG_BN) / ZG_THREADS; e++) {
            int idx = tid + e * ZG_THREADS, k = idx / ZG_BN, c = idx % ZG_BN;
            int gk = k0 + k, gc = col0 + c;
            bool ok = gk < p.K && gc < p.Nc;
            const cplx *src = ok ? B + (long long)gk * p.ldb + gc : B;
            cp_async16(dB + k * ZG_LDB + c, src, ok ? 16 : 0);
        }
        cp_async_commit();
    };

    double cre[4][4][2], cim[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) { cre[i][j][0] = cre[i][j][1] = 0.0; cim[i][j][0] = cim[i][j][1] = 0.0; }

    int mb_valid = (p.Mr - (row0 + wr) + 7) / 8; mb_valid = mb_valid < 0 ? 0 : (mb_valid > 4 ? 4 : mb_valid);
    int nb_valid = (p.Nc - (col0 + wc) + 7) / 8; nb_valid = nb_valid < 0 ? 0 : (nb_valid > 4 ? 4 : nb_valid);

    const double asign = p.conjA ? -1.0 : 1.0;
    const int nk = (p.K + ZG_BK - 1) / ZG_BK;
    load_stage(0, 0);
    for (int kt = 0; kt < nk; kt++) {
        if (kt + 1 < nk) { load_stage((kt + 1) & 1, (kt + 1) * ZG_BK); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncthreads();
        const cplx *cA = sA + (kt & 1) * ZG_BM * ZG_LDA + wr * ZG_LDA;
        const cplx *cB = sB + (kt & 1) * ZG_BK * ZG_LDB + wc;
#pragma unroll
        for (int kk = 0; kk < ZG_BK; kk += 4)
            warp_zmma_k4<4, 4>(cre, cim, cA, ZG_LDA, cB, ZG_LDB, kk, mb_valid, nb_valid, g, t, asign);
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) {
            int r = row0 + wr + i * 8 + g, c = col0 + wc + j * 8 + 2 * t;
            if (r < p.Mr) {
#pragma unroll
                for (int q = 0; q < 2; q++)
                    if (c + q < p.Nc) {
                        cplx v = cmake(cre[i][j][q], cim[i][j][q]);
                        C[(long long)r * p.ldc + c + q] = cmul(p.alpha, v);
                    }
            }
        }
}

}  // namespace rgf
