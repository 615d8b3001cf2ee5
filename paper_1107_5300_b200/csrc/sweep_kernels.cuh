// sweep_kernels.cuh -- the O(M^2) kernels of the sweep: fused assembly of A_i (rows A1+A3 of
// SURVEY.md 8a), compact start of the propagator, lead set-up/update kernels and the Gamma trace.
//
// Index conventions: batch item bz = d * n_E + e (device d, energy e).  Bond masks are bytes:
//   bond[d][i+1][j] = m'_i[j]  for i = -1..L-1 (vacancy-aware inter-slice bond i <-> i+1)
//   hop [d][i][j]   = 1 iff the intra-slice bond j <-> j+1 of slice i is alive
// S_i = { j : (i + j) even } = { 2r + (i & 1) }: atoms of slice i bonded to slice i + 1.
#pragma once
#include "rgf_common.cuh"

namespace rgf {

// A_i = z I - H_i - t^2 m'_{i-1} (.) g_{i-1} (.) m'_{i-1}  [- Sigma_L if i = 0] [- Sigma_R if i = L-1],
// written in place over g_{i-1} (Eq. 4 in the direct form; V = t diag(m) makes
// V g V a masked scale, never a GEMM -- BASELINE.json:north_star item 2).
__global__ void assemble_kernel(cplx *Gall, int M, int L, int i, int n_E, int bz0,
                                const double *energies, double eta, double t,
                                const double *onsite, const uint8_t *bond, const uint8_t *hop,
                                const cplx *gL, const cplx *gR)
{
    const int bl = blockIdx.y;                 // index inside the cohort (G is cohort-local)
    const int bz = bz0 + bl, d = bz / n_E, e = bz % n_E;
    const long long MM = (long long)M * M;
    cplx *G = Gall + (long long)bl * MM;
    const double *eps = onsite + ((long long)d * L + i) * M;
    const uint8_t *mprev = bond + ((long long)d * (L + 1) + i) * M;        // m'_{i-1}
    const uint8_t *mlast = bond + ((long long)d * (L + 1) + L) * M;        // m'_{L-1}
    const uint8_t *hp = hop + ((long long)d * L + i) * M;
    const double t2 = t * t;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < MM;
         idx += (long long)gridDim.x * blockDim.x) {
        int j = (int)(idx / M), k = (int)(idx % M);
        cplx a = cmake(0.0, 0.0);
        if (j == k) a = cmake(energies[e] - eps[j], eta);
        else if (k == j + 1) { if (hp[j]) a.x = -t; }
        else if (j == k + 1) { if (hp[k]) a.x = -t; }
        if (mprev[j] && mprev[k]) {
            // i = 0: previous "slice" is the left lead's surface slice -1
            cplx gp = (i == 0) ? gL[(long long)e * MM + idx] : G[idx];
            a.x -= t2 * gp.x; a.y -= t2 * gp.y;
        }
        if (i == L - 1 && mlast[j] && mlast[k]) {
            cplx gr = gR[(long long)e * MM + idx];
            a.x -= t2 * gr.x; a.y -= t2 * gr.y;
        }
        G[idx] = a;
    }
}

// ---- the sweep from the right end (rgf_api.cu: run_dense_two_sided) -------------------------------------------------
// gR_i = (z - H_i - t^2 m'_i (.) gR_{i+1} (.) m'_i)^-1, gR_L = surface Green's function of the right lead (Sigma_R at i = L-1):
// the mirror image of assemble_kernel, written in place over gR_{i+1}.  Used for slices i >= 1 only (no Sigma_L).
__global__ void assemble_right_kernel(cplx *Gall, int M, int L, int i, int n_E, int bz0, const double *energies, double eta, double t,
                                      const double *onsite, const uint8_t *bond, const uint8_t *hop, const cplx *gR)
{
    const int bl = blockIdx.y, bz = bz0 + bl, d = bz / n_E, e = bz % n_E;
    const long long MM = (long long)M * M;
    cplx *G = Gall + (long long)bl * MM;
    const double *eps = onsite + ((long long)d * L + i) * M;
    const uint8_t *mnext = bond + ((long long)d * (L + 1) + i + 1) * M;      // m'_i: bond between slices i and i + 1
    const uint8_t *hp = hop + ((long long)d * L + i) * M;
    const double t2 = t * t;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < MM; idx += (long long)gridDim.x * blockDim.x) {
        const int j = (int)(idx / M), k = (int)(idx % M);
        cplx a = cmake(0.0, 0.0);
        if (j == k) a = cmake(energies[e] - eps[j], eta);
        else if (k == j + 1) { if (hp[j]) a.x = -t; }
        else if (j == k + 1) { if (hp[k]) a.x = -t; }
        if (mnext[j] && mnext[k]) {
            const cplx g = (i == L - 1) ? gR[(long long)e * MM + idx] : G[idx];
            a.x -= t2 * g.x; a.y -= t2 * g.y;
        }
        G[idx] = a;
    }
}

// compact block of a full M x M matrix: Out[r][c] = G[2r + pr][2c + pc] (ld = nh), r < count(pr), c < count(pc)
__global__ void block_extract_kernel(const cplx *Gall, cplx *Out, int M, int nh, int pr, int pc)
{
    const int bl = blockIdx.y, nr = (M - pr + 1) / 2, ncol = (M - pc + 1) / 2;
    const cplx *G = Gall + (long long)bl * M * M;
    cplx *O = Out + (long long)bl * nh * nh;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < nr * ncol; idx += gridDim.x * blockDim.x) {
        const int r = idx / ncol, c = idx % ncol;
        O[(long long)r * nh + c] = G[(long long)(2 * r + pr) * M + 2 * c + pc];
    }
}

// P_0 = g_0 restricted to rows S_0 and columns S_{-1} (compact nh x nh storage, ld = nh).
__global__ void propagator_start_kernel(const cplx *Gall, cplx *Pall, int M, int nh)
{
    const int bl = blockIdx.y;
    const cplx *G = Gall + (long long)bl * M * M;
    cplx *P = Pall + (long long)bl * nh * nh;
    const int nr = (M + 1) / 2, nc = M / 2;      // |S_0| (even j), |S_{-1}| (odd j)
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < nr * nc; idx += gridDim.x * blockDim.x) {
        int r = idx / nc, c = idx % nc;
        P[(long long)r * nh + c] = G[(long long)(2 * r) * M + (2 * c + 1)];
    }
}

// ---- lead decimation (Sancho-Rubio on the clean two-slice cell): kernels in half_kernels.cuh ----
// alpha = h01 and beta = h01^T keep their block shape under alpha <- alpha g alpha, beta <- beta g beta (only block
// (2,1) resp. (1,2) of the 2M x 2M cell is ever non-zero, and inside it only the rows / columns of the atoms that bond to
// the next cell), so the products reduce to
//   alpha g beta = a g11 b on [2,2]      beta g alpha = b g22 a on [1,1]      alpha g alpha -> a g12 a      beta g beta -> b g21 b
// which are the dense products with their structurally-zero terms left out.

// flags[e] = 1 if max(|alpha|, |beta|) >= tol for energy e; *n_open counts them
__global__ void lead_converged_kernel(const cplx *alpha, const cplx *beta, int M, double tol, int *flags, int *n_open)
{
    const int e = blockIdx.x;
    const long long MM = (long long)M * M, off = (long long)e * MM;
    double m = 0.0;
    for (long long idx = threadIdx.x; idx < MM; idx += blockDim.x) {
        double a = cabs2(alpha[off + idx]), b = cabs2(beta[off + idx]);
        a = a > b ? a : b;
        if (!(a <= m)) m = a;          // NaN propagates as "not converged"
    }
    __shared__ double red[32];
    for (int o = 16; o > 0; o >>= 1) { double x = __shfl_xor_sync(0xffffffffu, m, o); if (!(x <= m)) m = x; }
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); w++) if (!(red[w] <= m)) m = red[w];
        int open = !(m < tol * tol);
        flags[e] = open;
        if (open) atomicAdd(n_open, 1);
    }
}

// ---- trace -------------------------------------------------------------
// Gamma = i (Sigma - Sigma^dagger) = -2 Im Sigma (Sigma is complex symmetric), Sigma = t^2 m (.) g (.) m.
// GamR compact on S_{L-1} x S_{L-1}: GamR[r][r'] = -2 t^2 m[jr] m[jr'] Im gR[e][jr][jr'], jr = 2r + pR.
__global__ void gamma_right_kernel(cplx *GamAll, const cplx *gR, const uint8_t *bond, int M, int L, int nh, int n_E, int bz0, double t)
{
    const int bl = blockIdx.y, bz = bz0 + bl, d = bz / n_E, e = bz % n_E;
    const int pR = (L - 1) & 1, nr = (M - pR + 1) / 2;
    const uint8_t *m = bond + ((long long)d * (L + 1) + L) * M;
    cplx *Gam = GamAll + (long long)bl * nh * nh;
    const cplx *g = gR + (long long)e * M * M;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < nr * nr; idx += gridDim.x * blockDim.x) {
        int r = idx / nr, c = idx % nr, jr = 2 * r + pR, jc = 2 * c + pR;
        double v = (m[jr] && m[jc]) ? -2.0 * t * t * g[(long long)jr * M + jc].y : 0.0;
        Gam[(long long)r * nh + c] = cmake(v, 0.0);
    }
}

// T = Re sum_{c,c'} GamL[c][c'] Y[c'][c],  Y = P^dagger GamR P (nc x nc, ld = nh), GamL real, on S_{-1} (odd j).
__global__ void trace_kernel(const cplx *Yall, const cplx *gL, const uint8_t *bond, int M, int L, int nh, int n_E, int bz0,
                             double t, double *T_out)
{
    const int bl = blockIdx.x, bz = bz0 + bl, d = bz / n_E, e = bz % n_E;
    const int nc = M / 2;
    const uint8_t *m = bond + ((long long)d * (L + 1) + 0) * M;    // m'_{-1}
    const cplx *Y = Yall + (long long)bl * nh * nh;
    const cplx *g = gL + (long long)e * M * M;
    double acc = 0.0;
    for (int idx = threadIdx.x; idx < nc * nc; idx += blockDim.x) {
        int c = idx / nc, c2 = idx % nc, j = 2 * c + 1, j2 = 2 * c2 + 1;
        if (m[j] && m[j2]) acc += (-2.0 * t * t * g[(long long)j * M + j2].y) * Y[(long long)c2 * nh + c].x;
    }
    __shared__ double red[32];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) T_out[bz] = v;
    }
}

// expand the compact propagator into a full M x M matrix (NaN where not propagated), for rgf_sweep_state
__global__ void propagator_expand_kernel(const cplx *Pall, cplx *Out, int M, int nh, int pi)
{
    const int bl = blockIdx.y;
    const cplx *P = Pall + (long long)bl * nh * nh;
    cplx *O = Out + (long long)bl * M * M;
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < M * M; idx += gridDim.x * blockDim.x) {
        int j = idx / M, k = idx % M;
        bool have = ((j & 1) == pi) && ((k & 1) == 1);
        O[idx] = have ? P[(long long)(j >> 1) * nh + (k >> 1)] : cmake(nan, nan);
    }
}

// failed batch items -> NaN: status per item (sweep), lead_flags / lead_status per energy (decimation not converged / bad pivot)
__global__ void fill_nan_kernel(double *T, const int *status, const int *lead_flags, const int *lead_status, int n, int n_E)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && (status[i] || lead_flags[i % n_E] || lead_status[i % n_E])) T[i] = __longlong_as_double(0x7ff8000000000000LL);
}

// guard: T_keep[d][idx[k]] = T2[d][k]
__global__ void scatter_T_kernel(double *T_keep, const double *T2, const int *idx, int n2, int n_E, int n_dev)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n2 * n_dev) T_keep[(long long)(i / n2) * n_E + idx[i % n2]] = T2[i];
}

}  // namespace rgf
