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

// ---- lead decimation on the corner blocks of the two-slice cell (rgf_api.cu: run_lead_side_schur) ---------------
// Compact nc x nc matrices, one per energy, contiguous: blocks over the corner atoms e (first slice) / o (second
// slice) of the cell, the atoms j = 2r + qc that bond to the neighbouring cells.

// a = b = t I; X = Y = S = 0
__global__ void lead_half_init_kernel(cplx *a, cplx *b, cplx *X, cplx *Y, cplx *Sacc, int nc, double t)
{
    const long long off = (long long)blockIdx.y * nc * nc;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < nc * nc; idx += gridDim.x * blockDim.x) {
        const cplx d = cmake((idx / nc == idx % nc) ? t : 0.0, 0.0), z = cmake(0.0, 0.0);
        a[off + idx] = d; b[off + idx] = d; X[off + idx] = z; Y[off + idx] = z; Sacc[off + idx] = z;
    }
}

// Schur complement of (z - eps) on the corner atoms (e, o), 2nc x 2nc, after the closed elimination of the pairs
// (f_j, b_j) of the other atoms:  S = [[z - Y - k1 K, -k2 K], [-k2 K, z - X - k1 K]], k1 = z / (z^2 - t^2),
// k2 = t / (z^2 - t^2), K[r][c] = t^2 * #(atoms adjacent to both corner atoms 2r+qc and 2c+qc).  X or Y may be NULL (= 0).
__global__ void lead_schur_assemble_kernel(cplx *Sall, const cplx *Xall, const cplx *Yall, int nc, int M, int qc, double t,
                                           const double *energies, double eta)
{
    const int e = blockIdx.y, N = 2 * nc;
    const long long NN = (long long)N * N, CC = (long long)nc * nc;
    cplx *S = Sall + (long long)e * NN;
    const cplx *X = Xall ? Xall + (long long)e * CC : nullptr, *Y = Yall ? Yall + (long long)e * CC : nullptr;
    const cplx z = cmake(energies[e], eta);
    const cplx den = crecip(cmake(z.x * z.x - z.y * z.y - t * t, 2.0 * z.x * z.y));       // 1 / (z^2 - t^2)
    const cplx k1 = cmul(z, den), k2 = cmake(t * den.x, t * den.y);
    const double t2 = t * t;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < NN; idx += (long long)gridDim.x * blockDim.x) {
        const int R = (int)(idx / N), C = (int)(idx % N), br = R >= nc, bc = C >= nc, r = R - br * nc, c = C - bc * nc;
        double k = 0.0;
        if (r == c) { const int j = 2 * r + qc; k = t2 * ((j - 1 >= 0 ? 1 : 0) + (j + 1 < M ? 1 : 0)); }
        else if (r == c + 1 || c == r + 1) k = t2;
        cplx v;
        if (br == bc) {
            v = cmake(-k * k1.x, -k * k1.y);
            if (r == c) { v.x += z.x; v.y += z.y; }
            const cplx *D = br ? X : Y;
            if (D) { const cplx d = D[(long long)r * nc + c]; v.x -= d.x; v.y -= d.y; }
        } else {
            v = cmake(-k * k2.x, -k * k2.y);
        }
        S[idx] = v;
    }
}

// X += sym(Tx); Y += sym(Ty); surface accumulator += sym(Tx) (right lead, side > 0: eps_s gets alpha g beta) or sym(Ty)
// (left lead).  With beta = alpha^T both increments are complex symmetric; averaging the two roundings keeps X, Y exactly
// symmetric, without which an antisymmetric rounding component doubles its exponent every iteration and the
// decimation diverges at some energies (seen at E = 0.4637 eV, M = 244).
__global__ void lead_half_accumulate_kernel(cplx *X, cplx *Y, cplx *Sacc, const cplx *Tx, const cplx *Ty, int nc, int side)
{
    const long long off = (long long)blockIdx.y * nc * nc;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < nc * nc; idx += gridDim.x * blockDim.x) {
        const int r = idx / nc, c = idx % nc;
        const long long tr = off + (long long)c * nc + r;
        const cplx tx = cmake(0.5 * (Tx[off + idx].x + Tx[tr].x), 0.5 * (Tx[off + idx].y + Tx[tr].y));
        const cplx ty = cmake(0.5 * (Ty[off + idx].x + Ty[tr].x), 0.5 * (Ty[off + idx].y + Ty[tr].y));
        X[off + idx] = cadd(X[off + idx], tx);
        Y[off + idx] = cadd(Y[off + idx], ty);
        Sacc[off + idx] = cadd(Sacc[off + idx], side > 0 ? tx : ty);
    }
}

// G <- (G + G^T) / 2 in place (N x N per energy): S is complex symmetric, so is its inverse; the pivoted elimination
// returns it symmetric only to rounding, and the antisymmetric part is what the decimation amplifies (measured against
// an 80-bit reference at M = 128: error of the surface Green's function 3.3e-10 without, 4.5e-11 with this step)
__global__ void lead_half_symmetrize_kernel(cplx *Gall, int N)
{
    cplx *G = Gall + (long long)blockIdx.y * N * N;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < (long long)N * N; idx += (long long)gridDim.x * blockDim.x) {
        const int r = (int)(idx / N), c = (int)(idx % N);
        if (c > r) {
            const cplx u = G[idx], v = G[(long long)c * N + r];
            const cplx m = cmake(0.5 * (u.x + v.x), 0.5 * (u.y + v.y));
            G[idx] = m; G[(long long)c * N + r] = m;
        }
    }
}

// One Newton step of the inverse, G <- G + G (I - S G), in two kernels around two products:
//   R <- I - R   (R = S G on entry)            G <- sym(G + D)   (D = G R on entry)
__global__ void lead_half_residual_kernel(cplx *Rall, int N)
{
    cplx *R = Rall + (long long)blockIdx.y * N * N;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < (long long)N * N; idx += (long long)gridDim.x * blockDim.x) {
        const cplx v = R[idx];
        R[idx] = cmake(((idx / N == idx % N) ? 1.0 : 0.0) - v.x, -v.y);
    }
}
__global__ void lead_half_correct_kernel(cplx *Gall, const cplx *Dall, int N)
{
    cplx *G = Gall + (long long)blockIdx.y * N * N;
    const cplx *D = Dall + (long long)blockIdx.y * N * N;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < (long long)N * N; idx += (long long)gridDim.x * blockDim.x) {
        const int r = (int)(idx / N), c = (int)(idx % N);
        if (c >= r) {
            const long long tr = (long long)c * N + r;
            const cplx m = cmake(0.5 * (G[idx].x + D[idx].x + G[tr].x + D[tr].x), 0.5 * (G[idx].y + D[idx].y + G[tr].y + D[tr].y));
            G[idx] = m; G[tr] = m;
        }
    }
}

// at = a^T (beta = alpha^T is kept structurally, never iterated on its own)
__global__ void lead_half_transpose_kernel(cplx *at, const cplx *a, int nc)
{
    const long long off = (long long)blockIdx.y * nc * nc;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < nc * nc; idx += gridDim.x * blockDim.x)
        at[off + (long long)(idx % nc) * nc + idx / nc] = a[off + idx];
}

// W = z - eps of the whole two-slice cell (2M x 2M per energy): eps = h00 + X on (o, o) + Y on (e, e),
// h00 = [[H_c, V_a], [V_a, H_c]], H_c = t on the first sub / super diagonal, V_a = t diag(m_pa); e = atoms 2r + qc of
// the first slice, o = atoms 2r + qc of the second.  X or Y may be NULL (= 0).
__global__ void lead_cell_assemble_kernel(cplx *Wall, const cplx *Xall, const cplx *Yall, int nc, int M, int qc, int pa, double t,
                                          const double *energies, double eta)
{
    const int e = blockIdx.y, N = 2 * M;
    const long long NN = (long long)N * N, CC = (long long)nc * nc;
    cplx *W = Wall + (long long)e * NN;
    const cplx *X = Xall ? Xall + (long long)e * CC : nullptr, *Y = Yall ? Yall + (long long)e * CC : nullptr;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < NN; idx += (long long)gridDim.x * blockDim.x) {
        const int R = (int)(idx / N), C = (int)(idx % N), br = R >= M, bc = C >= M, j = R - br * M, k = C - bc * M;
        cplx v = cmake(0.0, 0.0);
        if (br == bc) {
            if (j == k) v = cmake(energies[e], eta);
            else if (j == k + 1 || k == j + 1) v.x = -t;
            if ((j & 1) == qc && (k & 1) == qc) {
                const cplx *D = br ? X : Y;
                if (D) { const cplx d = D[(long long)(j >> 1) * nc + (k >> 1)]; v.x -= d.x; v.y -= d.y; }
            }
        } else if (j == k && mask_bit(pa, j)) {
            v.x = -t;
        }
        W[idx] = v;
    }
}

// surface Green's function on the coupled atoms j = 2r + qc: block of g with row stride ldg and column stride cs
// -> full M x M array (zeroed by the caller)
__global__ void lead_half_scatter_kernel(cplx *gfull, const cplx *G, int M, int nc, int qc, long long ldg, int cs, long long g_batch)
{
    const int e = blockIdx.y;
    const cplx *src = G + (long long)e * g_batch;
    cplx *dst = gfull + (long long)e * M * M;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < nc * nc; idx += gridDim.x * blockDim.x) {
        const int r = idx / nc, c = idx % nc;
        dst[(long long)(2 * r + qc) * M + 2 * c + qc] = src[(long long)r * ldg + (long long)c * cs];
    }
}

}  // namespace rgf
