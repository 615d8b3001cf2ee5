// ldos_kernels.cuh -- O(M^2) kernels of rgf_ldos: the diagonal blocks of the CONNECTED Green's function and the local
// density of states ("any desired quantity, e.g. charge density", PAPER.md:61 step 5).
//
// Two-sided form of the recursion (Eq. 3-4 applied from both ends; the oracle uses the other textbook form, the backward
// Dyson update G_ii = g_i + g_i V G_{i+1,i+1} V g_i, so the two share no formula beyond Eq. 1):
//   right-to-left   gR_i = (z - H_i - V_i gR_{i+1} V_i)^-1,  gR_L = surface Green's function of the right lead
//   left-to-right   gL_i = (z - H_i - V_{i-1} gL_{i-1} V_{i-1})^-1,  gL_{-1} = surface Green's function of the left lead
//                   G_ii = (z - H_i - V_{i-1} gL_{i-1} V_{i-1} - V_i gR_{i+1} V_i)^-1,   LDOS(i, j) = -(1/pi) Im G_ii[j][j]
// V_i = t diag(m'_i) keeps only the block of gR_{i+1} on S_i = { j : (i + j) even }, which is what is stashed between the
// two passes ((M/2)^2 elements per slice and matrix instead of M^2).  The inverses are the library's batched Gauss-Jordan.
// Scheduling (rgf_api.cu: rgf_ldos): the gR chain and the gL chain are sequential in i but independent of each other, so they
// run side by side on two streams, both stashing their blocks; the G_ii of ALL slices are then independent and are inverted
// in large batches of (matrix, slice) pairs -- latency-bound chains overlapped, the third inverse per slice throughput-bound.
#pragma once
#include "rgf_common.cuh"

namespace rgf {

// A (M x M per matrix) = z - H_i [- t^2 m'_{i-1} (.) gLeft (.) m'_{i-1}] [- t^2 m'_i (.) gRight (.) m'_i]
//   left  source: i == 0 ? lead surface gLlead[e] (full M x M) : gPrevFull[bl] (full M x M, the previous slice's gL)
//   right source: i == L-1 ? lead surface gRlead[e] (full)      : stashNext[bl] (compact block of gR_{i+1} on S_i, ld nh)
__global__ void ldos_assemble_kernel(cplx *Aall, int M, int L, int nh, int i, int n_E, int bz0, const double *energies, double eta, double t,
                                     const double *onsite, const uint8_t *bond, const uint8_t *hop, int use_left, const cplx *gPrevFull,
                                     const cplx *gLlead, int use_right, const cplx *stashNext, const cplx *gRlead)
{
    const int bl = blockIdx.y, bz = bz0 + bl, d = bz / n_E, e = bz % n_E;
    const long long MM = (long long)M * M;
    cplx *A = Aall + (long long)bl * MM;
    const double *eps = onsite + ((long long)d * L + i) * M;
    const uint8_t *mL = bond + ((long long)d * (L + 1) + i) * M;          // m'_{i-1}
    const uint8_t *mR = bond + ((long long)d * (L + 1) + i + 1) * M;      // m'_i
    const uint8_t *hp = hop + ((long long)d * L + i) * M;
    const double t2 = t * t;
    const int p = i & 1;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < MM; idx += (long long)gridDim.x * blockDim.x) {
        const int j = (int)(idx / M), k = (int)(idx % M);
        cplx a = cmake(0.0, 0.0);
        if (j == k) a = cmake(energies[e] - eps[j], eta);
        else if (k == j + 1) { if (hp[j]) a.x = -t; }
        else if (j == k + 1) { if (hp[k]) a.x = -t; }
        if (use_left && mL[j] && mL[k]) {
            const cplx g = (i == 0) ? gLlead[(long long)e * MM + idx] : gPrevFull[(long long)bl * MM + idx];
            a.x -= t2 * g.x; a.y -= t2 * g.y;
        }
        if (use_right && mR[j] && mR[k]) {
            const cplx g = (i == L - 1) ? gRlead[(long long)e * MM + idx]
                                        : stashNext[(long long)bl * nh * nh + (long long)((j - p) >> 1) * nh + ((k - p) >> 1)];
            a.x -= t2 * g.x; a.y -= t2 * g.y;
        }
        A[idx] = a;
    }
}

// stash[bl][r][c] = G[bl][2r + p][2c + p]: the block of gR_i that slice i - 1 couples to (p = parity of S_{i-1})
__global__ void ldos_stash_kernel(const cplx *Gall, cplx *stash, int M, int nh, int p)
{
    const int bl = blockIdx.y, n = (M - p + 1) / 2;
    const cplx *G = Gall + (long long)bl * M * M;
    cplx *S = stash + (long long)bl * nh * nh;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n * n; idx += gridDim.x * blockDim.x) {
        const int r = idx / n, c = idx % n;
        S[(long long)r * nh + c] = G[(long long)(2 * r + p) * M + 2 * c + p];
    }
}

// A for a BATCH of (matrix, slice) pairs, y = blockIdx.y = (i - i0) * nb + bl, both neighbours from the stashes:
//   A = z - H_i - t^2 m'_{i-1} (.) gL_{i-1} (.) m'_{i-1} - t^2 m'_i (.) gR_{i+1} (.) m'_i
//   gL_{i-1}: i == 0 ? lead surface (full) : stashL[i-1][bl] (compact block on S_{i-1});  gR_{i+1}: i == L-1 ? lead : stashR[i+1][bl]
__global__ void ldos_assemble_both_kernel(cplx *Aall, int M, int L, int nh, int i0, int nb, int n_E, int bz0, const double *energies, double eta,
                                          double t, const double *onsite, const uint8_t *bond, const uint8_t *hop, const cplx *stashL,
                                          const cplx *stashR, const cplx *gLlead, const cplx *gRlead)
{
    const int y = blockIdx.y, bl = y % nb, i = i0 + y / nb, bz = bz0 + bl, d = bz / n_E, e = bz % n_E;
    const long long MM = (long long)M * M, hs = (long long)nh * nh;
    cplx *A = Aall + (long long)y * MM;
    const double *eps = onsite + ((long long)d * L + i) * M;
    const uint8_t *mL = bond + ((long long)d * (L + 1) + i) * M;          // m'_{i-1}
    const uint8_t *mR = bond + ((long long)d * (L + 1) + i + 1) * M;      // m'_i
    const uint8_t *hp = hop + ((long long)d * L + i) * M;
    const cplx *sL = i > 0 ? stashL + ((long long)(i - 1) * nb + bl) * hs : nullptr;
    const cplx *sR = i < L - 1 ? stashR + ((long long)(i + 1) * nb + bl) * hs : nullptr;
    const double t2 = t * t;
    const int p = i & 1, q = 1 - p;                                        // parity of S_i and of S_{i-1}
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < MM; idx += (long long)gridDim.x * blockDim.x) {
        const int j = (int)(idx / M), k = (int)(idx % M);
        cplx a = cmake(0.0, 0.0);
        if (j == k) a = cmake(energies[e] - eps[j], eta);
        else if (k == j + 1) { if (hp[j]) a.x = -t; }
        else if (j == k + 1) { if (hp[k]) a.x = -t; }
        if (mL[j] && mL[k]) {
            const cplx g = sL ? sL[(long long)((j - q) >> 1) * nh + ((k - q) >> 1)] : gLlead[(long long)e * MM + idx];
            a.x -= t2 * g.x; a.y -= t2 * g.y;
        }
        if (mR[j] && mR[k]) {
            const cplx g = sR ? sR[(long long)((j - p) >> 1) * nh + ((k - p) >> 1)] : gRlead[(long long)e * MM + idx];
            a.x -= t2 * g.x; a.y -= t2 * g.y;
        }
        A[idx] = a;
    }
}

// out[bl][i][j] = -(1/pi) Im G[y][j][j], y = (i - i0) * nb + bl; a bad pivot of item y gives NaN and flags the matrix
__global__ void ldos_diag_kernel(const cplx *Gall, double *out, const int *dstat, int *status, int M, int L, int i0, int nb, int ns)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)nb * ns * M) return;
    const int y = (int)(idx / M), j = (int)(idx % M), bl = y % nb, i = i0 + y / nb;
    const double v = -Gall[(long long)y * M * M + (long long)j * M + j].y * 0.31830988618379067154;
    const bool bad = dstat[y] != 0;
    if (bad && j == 0) status[bl] = 1;
    out[((long long)bl * L + i) * M + j] = bad ? __longlong_as_double(0x7ff8000000000000LL) : v;
}

}  // namespace rgf
