// half_kernels.cuh -- O(M^2) kernels of the half-slice formulation of the sweep.
//
// The armchair slice i splits into two half-slices:
//   B_i = { j : (i + j) odd  }  atoms bonded backwards, to slice i - 1 (same j, hopping t m'_{i-1}[j])
//   F_i = { j : (i + j) even }  atoms bonded forwards,  to slice i + 1
// and inside the slice every bond j <-> j+1 joins one B atom and one F atom.  The recursion of
// PAPER.md:47-51 (Eq. 4-5) applied to the finer slicing ..., B_i, F_i, B_{i+1}, ... is
//   kind B:  gB_i = (z - eps_B - t^2 m' (.) gF_{i-1} (.) m')^-1          PB_i = gB_i (t m' (.) PF_{i-1})
//   kind F:  gF_i = (z - eps_F - C gB_i C^T [- Sigma_R if i = L-1])^-1   PF_i = gF_i (C PB_i)
// with C[f][b] = t hop[i][min(jf, jb)] for |jf - jb| = 1 (two entries per row: a stencil, never a
// GEMM).  gF_i equals the F x F block of the full-slice G_ii and PF_i the rows F_i of G_{i,0}.
// Compact index r of atom j with parity par: j = 2 r + par; count(par) = (M - par + 1) / 2.
// g matrices are dense n x n (ld = n) at batch stride nh*nh; P, W are n x (M/2) with ld = nh.
#pragma once
#include "rgf_common.cuh"

namespace rgf {

__host__ __device__ __forceinline__ int half_count(int M, int par) { return (M - par + 1) / 2; }

struct HalfArgs {
    int M, L, nh, i, kind;          // kind 0 = B half of slice i, 1 = F half
    int n_E, bz0;
    double eta, t;
    const double *energies, *onsite;
    const uint8_t *bond, *hop;
    const cplx *gL, *gR;            // lead surface Green's functions [n_E][M][M]
};

// neighbour s of F atom r (parity p) on side `up` (0: j-1, 1: j+1) in the B half (parity q = 1-p);
// returns -1 when the bond does not exist or is dead
__device__ __forceinline__ int half_nbr(int r, int p, int up, int M, const uint8_t *hp)
{
    const int j = 2 * r + p, jb = up ? j + 1 : j - 1;
    if (jb < 0 || jb >= M) return -1;
    if (!hp[up ? j : jb]) return -1;
    return (jb - (1 - p)) >> 1;
}

// A of the half-step, written to Aall (dense n x n, ld = n, batch stride nh*nh); gprev is the
// previous half-step's Green's function (dense nprev x nprev at the same stride).
__global__ void half_assemble_kernel(cplx *Aall, const cplx *gprev_all, HalfArgs a)
{
    const int bl = blockIdx.y, bz = a.bz0 + bl, d = bz / a.n_E, e = bz % a.n_E;
    const int M = a.M, L = a.L, i = a.i;
    const long long hs = (long long)a.nh * a.nh, MM = (long long)M * M;
    cplx *A = Aall + bl * hs;
    const cplx *gp = gprev_all + bl * hs;
    const double t2 = a.t * a.t, E = a.energies[e];
    const double *eps = a.onsite + ((long long)d * L + i) * M;
    if (a.kind == 0) {
        const int q = (i + 1) & 1, n = half_count(M, q);
        const uint8_t *mk = a.bond + ((long long)d * (L + 1) + i) * M;       // m'_{i-1}
        const cplx *gl = a.gL + (long long)e * MM;
        for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n * n; idx += gridDim.x * blockDim.x) {
            const int r = idx / n, c = idx % n, jr = 2 * r + q, jc = 2 * c + q;
            cplx v = cmake(0.0, 0.0);
            if (r == c) v = cmake(E - eps[jr], a.eta);
            if (mk[jr] && mk[jc]) {
                const cplx g = (i == 0) ? gl[(long long)jr * M + jc] : gp[idx];
                v.x -= t2 * g.x; v.y -= t2 * g.y;
            }
            A[idx] = v;
        }
    } else {
        const int p = i & 1, n = half_count(M, p), nb = half_count(M, 1 - p);
        const uint8_t *hp = a.hop + ((long long)d * L + i) * M;
        const uint8_t *mr = a.bond + ((long long)d * (L + 1) + L) * M;       // m'_{L-1}
        const cplx *gr = a.gR + (long long)e * MM;
        for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n * n; idx += gridDim.x * blockDim.x) {
            const int r = idx / n, c = idx % n;
            cplx v = cmake(0.0, 0.0);
            if (r == c) v = cmake(E - eps[2 * r + p], a.eta);
            double sx = 0.0, sy = 0.0;
#pragma unroll
            for (int u = 0; u < 2; u++) {
                const int sr = half_nbr(r, p, u, M, hp);
                if (sr < 0) continue;
#pragma unroll
                for (int w = 0; w < 2; w++) {
                    const int sc = half_nbr(c, p, w, M, hp);
                    if (sc < 0) continue;
                    const cplx g = gp[(long long)sr * nb + sc];
                    sx += g.x; sy += g.y;
                }
            }
            v.x -= t2 * sx; v.y -= t2 * sy;
            if (i == L - 1) {
                const int jr = 2 * r + p, jc = 2 * c + p;
                if (mr[jr] && mr[jc]) { const cplx g = gr[(long long)jr * M + jc]; v.x -= t2 * g.x; v.y -= t2 * g.y; }
            }
            A[idx] = v;
        }
    }
}

// W = C P_prev (rows of the new half-step, nc columns, ld = nh).  Kind B of slice 0 has no
// previous propagator: P = gB_0 itself is written by half_start_kernel instead.
__global__ void half_couple_kernel(cplx *Wall, const cplx *Pall, HalfArgs a)
{
    const int bl = blockIdx.y, bz = a.bz0 + bl, d = bz / a.n_E;
    const int M = a.M, L = a.L, i = a.i, nh = a.nh, nc = M / 2;
    const long long hs = (long long)nh * nh;
    cplx *W = Wall + bl * hs;
    const cplx *P = Pall + bl * hs;
    if (a.kind == 0) {
        const int q = (i + 1) & 1, n = half_count(M, q);
        const uint8_t *mk = a.bond + ((long long)d * (L + 1) + i) * M;
        for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n * nc; idx += gridDim.x * blockDim.x) {
            const int r = idx / nc, c = idx % nc;
            const double s = mk[2 * r + q] ? a.t : 0.0;
            const cplx v = P[(long long)r * nh + c];
            W[(long long)r * nh + c] = cmake(s * v.x, s * v.y);
        }
    } else {
        const int p = i & 1, n = half_count(M, p);
        const uint8_t *hp = a.hop + ((long long)d * L + i) * M;
        for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n * nc; idx += gridDim.x * blockDim.x) {
            const int r = idx / nc, c = idx % nc;
            double sx = 0.0, sy = 0.0;
#pragma unroll
            for (int u = 0; u < 2; u++) {
                const int s = half_nbr(r, p, u, M, hp);
                if (s >= 0) { const cplx v = P[(long long)s * nh + c]; sx += v.x; sy += v.y; }
            }
            W[(long long)r * nh + c] = cmake(a.t * sx, a.t * sy);
        }
    }
}

// PB_0 = gB_0 (rows B_0 = odd j, columns B_0): dense n x n (ld n) -> ld nh
__global__ void half_start_kernel(cplx *Pall, const cplx *gall, int n, int nh)
{
    const int bl = blockIdx.y;
    const long long hs = (long long)nh * nh;
    cplx *P = Pall + bl * hs;
    const cplx *g = gall + bl * hs;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n * n; idx += gridDim.x * blockDim.x)
        P[(long long)(idx / n) * nh + idx % n] = g[idx];
}

// for rgf_sweep_state: gF (n x n, ld n) -> full M x M with NaN outside F x F
__global__ void half_expand_g_kernel(const cplx *gall, cplx *Out, int M, int nh, int p)
{
    const int bl = blockIdx.y, n = half_count(M, p);
    const cplx *g = gall + (long long)bl * nh * nh;
    cplx *O = Out + (long long)bl * M * M;
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < M * M; idx += gridDim.x * blockDim.x) {
        const int j = idx / M, k = idx % M;
        const bool have = ((j & 1) == p) && ((k & 1) == p);
        O[idx] = have ? g[(long long)(j >> 1) * n + (k >> 1)] : cmake(nan, nan);
    }
}

}  // namespace rgf
