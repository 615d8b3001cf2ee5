// half_sweep_la.cuh -- fused half-slice sweep with panel look-ahead: ONE CTA of 16 warps per SM and per matrix.
//
// Same recursion, same augmented Gauss-Jordan and the same device functions as half_sweep.cuh (Eq. 4-5
// on the slicing B_0, F_0, B_1, ...); what differs is who does what, and when:
//   * warps 0-3 ("factor warps", one per SM sub-partition, thread = row) own the serial pivot chain.  While panel p is
//     being applied they first update the four 8-column strips that hold panel p+1, then load and factor panel p+1
//     in the second panel buffer;
//   * warps 4-15 ("update warps") apply panel p to every other strip of [X | W] on the FP64 tensor pipe (barrier-free
//     strips, hs_strip_update), so the pivot chain of panel p+1 runs under the DMMAs of panel p;
//   * only the assembly, the first panel of a half-step and the last update have no partner.
// One matrix per SM instead of two halves the live state (148 x 0.95 MB), so the active buffers of all resident
// matrices (70 MB) stay in the 126 MB L2 instead of streaming through HBM.
#pragma once
#include "half_sweep.cuh"

namespace rgf {

constexpr int LA_NT = 512, LA_NF = 128;          // threads per CTA, threads of the factor group
constexpr int LA_RB = 32;                        // output rows per staging block of the assembly

struct HSmemLA {
    cplx panel[2][HS_NMAX * HS_LDP];             // panel p (Mult) and panel p+1 (being factored); staging area of the assembly
    cplx Rs[HS_SB * HS_LDR];
    cplx crow[2 * (HS_NT / 32) * HS_SB];
    cplx cinv[2 * (HS_NT / 32)];
    alignas(16) unsigned ckey[2 * (HS_NT / 32)];
    int perm[HS_NMAX], pinv[HS_NMAX], perm_prev[HS_NMAX], pinv_prev[HS_NMAX];
    int prow[2][HS_B];
    long long prof[16];
};
static_assert(2 * (LA_RB + 2) * HS_NMAX <= 2 * HS_NMAX * HS_LDP, "two staging areas must fit in the panel buffers");

// panel columns [k0, k0 + bw) of X -> shared memory, by the factor group (cp.async.cg: L2, never a stale L1 line)
__device__ __forceinline__ void la_load_panel(cplx *panel, const cplx *X, int ld, int n, int k0, int bw)
{
    for (int e = threadIdx.x; e < HS_NMAX * HS_B; e += LA_NF) {
        const int rr = e / HS_B, c = e % HS_B;
        const bool ok = rr < n && c < bw;
        cp_async16(panel + rr * HS_LDP + c, ok ? X + (long long)rr * ld + k0 + c : X, ok ? 16 : 0);
    }
    cp_async_commit();
    cp_async_wait<0>();
    hs_bar(2, LA_NF);
}

__device__ __forceinline__ void la_strip(const cplx *panel, const int *prow, cplx *Cg, int ld, int n, int col0, int ncols, int bw)
{
    if (bw == HS_B) hs_strip_update<HS_RG, true>(panel, prow, Cg, ld, n, col0, ncols, bw);
    else hs_strip_update<HS_RG, false>(panel, prow, Cg, ld, n, col0, ncols, bw);
}

// ---- [X | W] <- A^-1 [I | W] in place (X holds A on entry); fills sm.perm / sm.pinv ------------------------
__device__ __forceinline__ void la_gauss_jordan(HSmemLA &sm, cplx *X, cplx *W, int ld, int n, int nc, int *status_slot, long long *prof)
{
    long long tc = prof ? clock64() : 0;
#define LA_TICK(slot) do { if (prof) { long long now_ = clock64(); if (threadIdx.x == 0) sm.prof[slot] += now_ - tc; tc = now_; } } while (0)
    const int tid = threadIdx.x, warp = tid >> 5;
    const bool isF = warp < LA_NF / 32;
    bool used = !(tid < n);
    HSGroup grp;
    grp.r = tid; grp.slot = warp; grp.nslots = (n + 31) >> 5; grp.gtid = tid; grp.gnt = LA_NF;
    grp.bar_pivot = 1; grp.n_pivot = grp.nslots * 32; grp.bar_all = 2;
    grp.rbase = warp * 32; grp.nbsel = 0; grp.nbmod = 1;
    HSView view;
    view.Rs = sm.Rs; view.crow = sm.crow; view.cinv = sm.cinv; view.ckey = sm.ckey;
    view.perm = sm.perm; view.pinv = sm.pinv; view.prof = nullptr;
    const int np = (n + HS_B - 1) / HS_B;
    const int nsx = (n + 7) >> 3, nsw = (nc + 7) >> 3;
    // first panel: nothing to overlap it with
    if (isF) {
        const int bw0 = n < HS_B ? n : HS_B;
        la_load_panel(sm.panel[0], X, ld, n, 0, bw0);
        view.panel = sm.panel[0]; view.prow = sm.prow[0];
        hs_factor_panel(view, grp, n, 0, bw0, used, status_slot);
    }
    __syncthreads();
    LA_TICK(2);
    for (int p = 0; p < np; p++) {
        const int cur = p & 1, k0 = p * HS_B, bw = (n - k0 < HS_B) ? (n - k0) : HS_B;
        cplx *panel = sm.panel[cur];
        const int *prow = sm.prow[cur];
        // N' -> X[:, K];  then the panel becomes Mult = N' - E (E[prow[c]][c] = 1)
        for (int e = tid; e < n * HS_B; e += LA_NT) {
            const int rr = e / HS_B, c = e % HS_B;
            if (c < bw) X[(long long)rr * ld + k0 + c] = panel[rr * HS_LDP + c];
        }
        __syncthreads();
        if (tid < bw) panel[prow[tid] * HS_LDP + tid].x -= 1.0;
        __syncthreads();
        LA_TICK(3);
        const bool more = p + 1 < np;
        const int sk0 = k0 >> 3;
        const int sk1 = (sk0 + HS_B / 8 < nsx) ? sk0 + HS_B / 8 : nsx;                    // strips of panel p: [sk0, sk1)
        const int sn1 = more ? ((sk1 + HS_B / 8 < nsx) ? sk1 + HS_B / 8 : nsx) : sk1;     // strips of panel p+1: [sk1, sn1)
        if (more && isF) {
            const int s = sk1 + warp;
            if (s < sn1) la_strip(panel, prow, X, ld, n, s * 8, n, bw);
            hs_bar(2, LA_NF);
            const int k1 = k0 + HS_B, bw1 = (n - k1 < HS_B) ? (n - k1) : HS_B;
            la_load_panel(sm.panel[cur ^ 1], X, ld, n, k1, bw1);
            view.panel = sm.panel[cur ^ 1]; view.prow = sm.prow[cur ^ 1];
            hs_factor_panel(view, grp, n, k1, bw1, used, status_slot);
        } else {
            // every other strip of X, then the strips of W, over the update warps (all warps behind the last panel)
            const int nw = more ? (LA_NT - LA_NF) / 32 : LA_NT / 32, w0 = more ? warp - LA_NF / 32 : warp;
            const int nxs = nsx - (sn1 - sk0), tot = nxs + nsw;
            for (int s = w0; s < tot; s += nw) {
                if (s < nxs) la_strip(panel, prow, X, ld, n, (s < sk0 ? s : s + (sn1 - sk0)) * 8, n, bw);
                else la_strip(panel, prow, W, ld, n, (s - nxs) * 8, nc, bw);
            }
        }
        __syncthreads();
        LA_TICK(4);
    }
#undef LA_TICK
}

// ---- the sweep: one CTA per matrix, half-steps [hs_begin, hs_end) of unit (matrix, chunk) ---------------------
__global__ void __launch_bounds__(LA_NT, 1) half_sweep_la_kernel(HSweepArgs a)
{
    extern __shared__ __align__(16) unsigned char hs_smem_raw[];
    HSmemLA &sm = *reinterpret_cast<HSmemLA *>(hs_smem_raw);
    const int tid = threadIdx.x, M = a.M, ld = a.ldn, nc = M / 2;
    const long long unit = (long long)a.unit0 + blockIdx.x;
    const int bl = (int)(unit % a.nb);
    const int hs_begin = a.hs_begin + (int)(unit / a.nb) * a.unit_len;
    const int hs_end = (hs_begin + a.unit_len < a.hs_end) ? hs_begin + a.unit_len : a.hs_end;
    if (hs_begin >= hs_end) return;
    const long long xs = (long long)ld * ld;
    cplx *const X0 = a.X0 + bl * xs, *const X1 = a.X1 + bl * xs, *const W0 = a.P0 + bl * xs, *const W1 = a.P1 + bl * xs;
    int *gperm = a.perm + (long long)bl * HS_NMAX;
    int *status_slot = a.status + bl;
    if (hs_begin > 0) {
        if (tid < HS_NMAX) sm.perm[tid] = gperm[tid];
        __syncthreads();
        const int hp_ = hs_begin - 1, ip = hp_ >> 1, kp = hp_ & 1;
        const int np = half_count(M, kp == 0 ? ((ip + 1) & 1) : (ip & 1));
        if (tid < np) sm.pinv[sm.perm[tid]] = tid;
        __syncthreads();
    }
    if (tid < 16) sm.prof[tid] = 0;
    const HSAsm av = {&sm.panel[0][0], reinterpret_cast<HSTab *>(sm.crow), sm.perm_prev, sm.pinv_prev};
    int n = 0;
    for (int hs = hs_begin; hs < hs_end; hs++) {
        const int i = hs >> 1, kind = hs & 1;
        cplx *Xp = kind ? X1 : X0, *Wp = kind ? W1 : W0, *Xn = kind ? X0 : X1, *Wn = kind ? W0 : W1;
        if (tid < HS_NMAX) { sm.perm_prev[tid] = sm.perm[tid]; sm.pinv_prev[tid] = sm.pinv[tid]; }
        __syncthreads();
        long long tc0 = a.prof ? clock64() : 0;
        hs_assemble<LA_NT, LA_RB>(av, a, bl, i, kind, hs == 0, Xp, Wp, Xn, Wn);
        __syncthreads();
        if (a.prof && tid == 0) sm.prof[0] += clock64() - tc0;
        n = half_count(M, kind == 0 ? ((i + 1) & 1) : (i & 1));
        la_gauss_jordan(sm, Xn, Wn, ld, n, nc, status_slot, a.prof ? a.prof + bl * 16 : nullptr);
    }
    if (tid < HS_NMAX) gperm[tid] = sm.perm[tid];
    if (a.prof && tid < 16) a.prof[bl * 16 + tid] += sm.prof[tid];
    if (hs_end == a.hs_end && (a.g_out || a.P_out)) {
        const cplx *Xf = (hs_end & 1) ? X1 : X0, *Wf = (hs_end & 1) ? W1 : W0;      // buffers written by the last half-step
        const long long os = (long long)a.nh * a.nh;
        if (a.g_out)
            for (int idx = tid; idx < n * n; idx += LA_NT) {
                const int k = idx / n, m = idx % n;
                a.g_out[bl * os + idx] = ldcg(Xf + (long long)sm.perm[k] * ld + sm.pinv[m]);
            }
        if (a.P_out)
            for (int idx = tid; idx < n * nc; idx += LA_NT) {
                const int k = idx / nc, c = idx % nc;
                a.P_out[bl * os + (long long)k * a.nh + c] = ldcg(Wf + (long long)sm.perm[k] * ld + c);
            }
    }
}

}  // namespace rgf
