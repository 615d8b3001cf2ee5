// lead_modes.cuh -- lead surface Green's function in transverse mode space (the paper's own
// route, "self-energies due to the leads which requires solution of an eigen-problem").
//
// The clean lead (H_c = t on the first sub / super diagonal, V_i = t diag(m_i), m_i[j] = 1 iff (i + j) even) is
// diagonal in the sine basis u_p[j] = sqrt(2/(M+1)) sin(p pi (j+1)/(M+1)), p = 1..M:
//     U^T H_c U = diag(2 t cos theta_p),   U^T diag((-1)^j) U = J  (J swaps p <-> M+1-p),   so  U^T V_i U = t (1 + (-1)^i J) / 2.
// In the combinations s_p = (u_p + u_p')/sqrt2 (supported on even j) and a_p = (u_p - u_p')/sqrt2 (odd j), p' = M+1-p,
// p = 1..M/2, slice i holds the two orbitals (s_p, a_p) joined by the hopping eps_p = 2 t cos theta_p, and consecutive
// slices are joined by t through s (i even) or a (i odd): every pair is ONE linear chain with alternating hoppings
// eps_p, t, eps_p, t, ...  The device couples to the end site of that chain (a_p of slice -1 on the left; s_p or a_p of
// slice L on the right), whose first bond into the lead is eps_p.  Its surface Green's function solves
//     G = 1 / (z - h1^2 / (z - h2^2 G)),   h1 = eps_p, h2 = t      (two decimation steps map the chain onto itself)
//     z h2^2 G^2 - (z^2 - h1^2 + h2^2) G + z = 0,   G = 2 z / (B +- sqrt(D)),   B = z^2 - h1^2 + h2^2,
//     D = (z - h1 - h2)(z + h1 + h2)(z - h1 + h2)(z + h1 - h2)       (product form: no cancellation at the band edges)
// and the retarded root is the attractive fixed point of the map (|f'(G)| < 1).  For odd M the middle mode p = (M+1)/2
// (eps = 0, J = +1) lives on even j and is an isolated site at the surface: G = 1 / z.
// On the atoms j = 2 r + qc of the surface slice that bond to the device the surface Green's function is
//     g[r][c] = sum_p Q[r][p] Q[c][p] G_p,     Q[r][p] = sqrt2 u_p[2 r + qc]     (Q is an orthogonal nc x nc matrix)
// O(M) closed forms + one real x complex product per energy; no iteration, no inverse, no resonance of the isolated
// cell (the Sancho-Rubio routes lose digits at |E - E_cell| -> 0).
#pragma once
#include "rgf_common.cuh"

namespace rgf {

// Q[r][p], r, p < nc (row-major).  Pair modes p = 0..M/2-1 (mode number p + 1); for odd M and qc = 0 the last column is
// the middle mode.  The argument of the sine is reduced in integers, so sinpi sees an exact rational.
__global__ void lead_modes_basis_kernel(double *Q, int M, int nc, int qc)
{
    const int np = M / 2;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < nc * nc; idx += gridDim.x * blockDim.x) {
        const int r = idx / nc, p = idx % nc, j = 2 * r + qc;
        double v;
        if (p < np) {
            const long long k = ((long long)(p + 1) * (j + 1)) % (2LL * (M + 1));
            v = 2.0 * rsqrt((double)(M + 1)) * sinpi((double)k / (double)(M + 1));
        } else {
            v = sqrt(2.0 / (double)(M + 1)) * sinpi(0.5 * (double)((j + 1) & 3));
        }
        Q[idx] = v;
    }
}

__device__ __forceinline__ cplx lm_csqrt(cplx a)
{
    const double m = hypot(a.x, a.y);
    if (m == 0.0) return cmake(0.0, 0.0);
    if (a.x >= 0.0) {
        const double re = sqrt(0.5 * (m + a.x));
        return cmake(re, 0.5 * a.y / re);
    }
    const double im = sqrt(0.5 * (m - a.x));
    return cmake(0.5 * fabs(a.y) / im, a.y >= 0.0 ? im : -im);
}

// surface Green's function of the end site of the semi-infinite chain with hoppings h1, h2, h1, ... at z (Im z > 0)
__device__ __forceinline__ cplx lm_chain_surface(cplx z, double h1, double h2)
{
    if (h1 == 0.0) return crecip(z);
    const cplx z2 = cmul(z, z);
    const cplx B = cmake(z2.x - h1 * h1 + h2 * h2, z2.y);
    cplx D = cmul(cmake(z.x - h1 - h2, z.y), cmake(z.x + h1 + h2, z.y));
    D = cmul(D, cmul(cmake(z.x - h1 + h2, z.y), cmake(z.x + h1 - h2, z.y)));
    const cplx s = lm_csqrt(D);
    cplx best = cmake(0.0, 0.0);
    double bd = 1e300;
#pragma unroll
    for (int k = 0; k < 2; k++) {
        const cplx den = k == 0 ? cadd(B, s) : csub(B, s);
        if (den.x == 0.0 && den.y == 0.0) continue;
        const cplx G = cmul(cmake(2.0 * z.x, 2.0 * z.y), crecip(den));
        // |f'(G)| = |G h1 h2 / (z - h2^2 G)|^2
        const cplx w = cmul(cmake(G.x * h1 * h2, G.y * h1 * h2), crecip(cmake(z.x - h2 * h2 * G.x, z.y - h2 * h2 * G.y)));
        const double d = cabs2(w);
        if (d < bd) { bd = d; best = G; }
    }
    return best;
}

// g_out[e][2r+qc][2c+qc] = sum_p Q[r][p] Q[c][p] G_p(z_e); the rest of g_out [n_E][M][M] is zeroed by the caller.
// 16 x 16 output tile per CTA, modes in chunks of 32 staged in shared memory.
__global__ void __launch_bounds__(256) lead_modes_kernel(cplx *g_out, const double *Q, int M, int nc, int qc, double t,
                                                         const double *energies, double eta)
{
    __shared__ double qa[16][33], qb[16][33];
    __shared__ cplx G0[32];
    const int e = blockIdx.z, r0 = blockIdx.y * 16, c0 = blockIdx.x * 16;
    const int tid = threadIdx.x, tr = tid >> 4, tc = tid & 15, np = M / 2;
    const cplx z = cmake(energies[e], eta);
    double ax = 0.0, ay = 0.0;
    for (int p0 = 0; p0 < nc; p0 += 32) {
        if (tid < 32) {
            const int p = p0 + tid;
            cplx G = cmake(0.0, 0.0);
            if (p < nc) {
                const long long k = (long long)(p + 1) % (2LL * (M + 1));
                const double h1 = p < np ? 2.0 * t * cospi((double)k / (double)(M + 1)) : 0.0;
                G = lm_chain_surface(z, h1, t);
            }
            G0[tid] = G;
        }
        for (int k = tid; k < 16 * 32; k += 256) {
            const int rr = k >> 5, pp = k & 31;
            qa[rr][pp] = (r0 + rr < nc && p0 + pp < nc) ? Q[(long long)(r0 + rr) * nc + p0 + pp] : 0.0;
            qb[rr][pp] = (c0 + rr < nc && p0 + pp < nc) ? Q[(long long)(c0 + rr) * nc + p0 + pp] : 0.0;
        }
        __syncthreads();
#pragma unroll 8
        for (int pp = 0; pp < 32; pp++) {
            const double w = qa[tr][pp] * qb[tc][pp];
            ax = fma(w, G0[pp].x, ax);
            ay = fma(w, G0[pp].y, ay);
        }
        __syncthreads();
    }
    const int r = r0 + tr, c = c0 + tc;
    if (r < nc && c < nc) g_out[(long long)e * M * M + (long long)(2 * r + qc) * M + 2 * c + qc] = cmake(ax, ay);
}

// Sigma = t^2 m (.) g (.) m for rgf_lead_self_energy (the same masked scale the sweep's assembly applies)
__global__ void lead_sigma_kernel(cplx *Sig, const cplx *g, const uint8_t *m, int M, double t)
{
    const long long MM = (long long)M * M, off = (long long)blockIdx.y * MM;
    const double t2 = t * t;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < MM; idx += (long long)gridDim.x * blockDim.x) {
        const int j = (int)(idx / M), k = (int)(idx % M);
        const double s = (m[j] && m[k]) ? t2 : 0.0;
        const cplx v = g[off + idx];
        Sig[off + idx] = cmake(s * v.x, s * v.y);
    }
}

}  // namespace rgf
