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

#ifndef LA_FSMSP
#define LA_FSMSP 1
#endif
#ifndef LA_NT_
#define LA_NT_ 512
#endif
constexpr int LA_NT = LA_NT_, LA_NF = 128;       // threads per CTA, threads of the factor group
constexpr int LA_U0 = LA_FSMSP ? 32 : LA_NF;        // first update thread (profiling)
constexpr int LA_RB = 32;                        // output rows per staging block of the assembly

struct HSmemLA {
    cplx panel[2][HS_NMAX * HS_LDP];             // panel p (Mult) and panel p+1 (being factored); staging area of the assembly
    cplx Rs[HS_SB * HS_LDR];
    cplx crow[2 * (HS_NT / 32) * HS_SB];
    cplx cinv[2 * (HS_NT / 32)];
    alignas(16) unsigned ckey[2 * (HS_NT / 32)];
    int perm[HS_NMAX], pinv[HS_NMAX], perm_prev[HS_NMAX], pinv_prev[HS_NMAX];
    int prow[2][HS_B];
    int next;                                    // next strip of the current update (dynamic distribution over the warps)
    HSTab tab;                                   // tables of the assembly (W is assembled while panel 0 is factored)
    long long prof[16];
};
static_assert(2 * (LA_RB + 2) * HS_NMAX <= 2 * HS_NMAX * HS_LDP, "two staging areas must fit in the panel buffers");

// panel columns [k0, k0 + bw) of X -> shared memory, by the factor group (cp.async.cg: L2, never a stale L1 line)
__device__ __forceinline__ void la_load_panel(cplx *panel, const cplx *X, int ld, int n, int k0, int bw, int ftid)
{
    for (int e = ftid; e < HS_NMAX * HS_B; e += LA_NF) {
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
// wfn() is run by the update warps while the factor warps factor the first panel (the assembly of W, which no one
// needs before the first update).
template <class WFn>
__device__ __forceinline__ void la_gauss_jordan(HSmemLA &sm, cplx *X, cplx *W, int ld, int n, int nc, int *status_slot, long long *prof, WFn &&wfn)
{
    long long tc = prof ? clock64() : 0;
#define LA_TICK(slot) do { if (prof) { long long now_ = clock64(); if (threadIdx.x == 0) sm.prof[slot] += now_ - tc; tc = now_; } } while (0)
    const int tid = threadIdx.x, warp = tid >> 5;
#if LA_FSMSP
    // factor warps = warps 0, 4, 8, 12: all on SM sub-partition 0 (warp id mod 4), which then runs no update warp while
    // a panel is factored.  A DFMA that competes with two or more warps streaming DMMAs on its sub-partition is starved
    // (measured: 8 -> 82 cycles per dependent DFMA beside one such warp, > 30 000 beside two), so the pivot chain must
    // not share a sub-partition with the updates.
    const bool isF = (warp & 3) == 0;
    const int fslot = warp >> 2, ftid = (fslot << 5) | (tid & 31);
    const int utid = ((warp >> 2) * 3 + (warp & 3) - 1) * 32 + (tid & 31);       // index among the update threads
#else
    const bool isF = warp < LA_NF / 32;
    const int fslot = warp, ftid = tid;
    const int utid = tid - LA_NF;
#endif
    bool used = !(ftid < n);
    HSGroup grp;
    grp.r = ftid; grp.slot = fslot; grp.nslots = (n + 31) >> 5; grp.gtid = ftid; grp.gnt = LA_NF;
    grp.bar_pivot = 1; grp.n_pivot = grp.nslots * 32; grp.bar_all = 2;
    grp.rbase = fslot * 32; grp.nbsel = 0; grp.nbmod = 1;
    HSView view;
    view.Rs = sm.Rs; view.crow = sm.crow; view.cinv = sm.cinv; view.ckey = sm.ckey;
    view.perm = sm.perm; view.pinv = sm.pinv; view.prof = prof ? sm.prof : nullptr;
    const int np = (n + HS_B - 1) / HS_B;
    const int nsx = (n + 7) >> 3, nsw = (nc + 7) >> 3;
    // first panel: only the assembly of W runs beside it
    if (isF) {
        const int bw0 = n < HS_B ? n : HS_B;
        la_load_panel(sm.panel[0], X, ld, n, 0, bw0, ftid);
        view.panel = sm.panel[0]; view.prow = sm.prow[0];
        hs_factor_panel<HS_FSB>(view, grp, n, 0, bw0, used, status_slot);
    } else {
        wfn(utid);
    }
    __syncthreads();
    LA_TICK(2);
    for (int p = 0; p < np; p++) {
        const int cur = p & 1, k0 = p * HS_B, bw = (n - k0 < HS_B) ? (n - k0) : HS_B;
        cplx *panel = sm.panel[cur];
        const int *prow = sm.prow[cur];
        const bool more = p + 1 < np;
        const int sk0 = k0 >> 3;
        const int sk1 = (sk0 + HS_B / 8 < nsx) ? sk0 + HS_B / 8 : nsx;                    // strips of panel p: [sk0, sk1)
        const int sn1 = more ? ((sk1 + HS_B / 8 < nsx) ? sk1 + HS_B / 8 : nsx) : sk1;     // strips of panel p+1: [sk1, sn1)
        // N' -> X[:, K];  then the panel becomes Mult = N' - E (E[prow[c]][c] = 1)
        for (int e = tid; e < n * HS_B; e += LA_NT) {
            const int rr = e / HS_B, c = e % HS_B;
            if (c < bw) X[(long long)rr * ld + k0 + c] = panel[rr * HS_LDP + c];
        }
        __syncthreads();
        if (tid < bw) panel[prow[tid] * HS_LDP + tid].x -= 1.0;      // (any bw threads)
        if (tid == 0) sm.next = 0;
        long long tq = prof ? clock64() : 0;
#define LA_TOCK(slot, who) do { if (prof) { long long now_ = clock64(); if (threadIdx.x == (who)) { sm.prof[slot] += now_ - tq; tq = now_; } } } while (0)
        if (more) {
            // the strips that hold panel p+1 come first, split over all 16 warps (strip = warp & 3, 32 rows each): every
            // warp reads its strip's pivot rows before the barrier, writes after it
            constexpr int PARTS = LA_NT / 128, RPP = ((HS_NMAX / PARTS + 15) / 16) * 16;
            const int s = sk1 + (warp & 3), r_begin = (warp >> 2) * RPP, nlim = (r_begin + RPP < n) ? r_begin + RPP : n;
            const bool act = s < sn1 && r_begin < n;
            cplx bb[8];
            if (act) hs_strip_load_b(bb, prow, X, ld, s * 8, n, bw);
            __syncthreads();
            if (act) {
                if (bw == HS_B) hs_strip_rows<HS_RG, true>(panel, bb, X, ld, r_begin, nlim, s * 8, n, bw);
                else hs_strip_rows<HS_RG, false>(panel, bb, X, ld, r_begin, nlim, s * 8, n, bw);
            }
        }
        __syncthreads();
        LA_TICK(3);
        LA_TOCK(12, 0);
        if (more && isF) {
            const int k1 = k0 + HS_B, bw1 = (n - k1 < HS_B) ? (n - k1) : HS_B;
            la_load_panel(sm.panel[cur ^ 1], X, ld, n, k1, bw1, ftid);
            LA_TOCK(6, 0);
            view.panel = sm.panel[cur ^ 1]; view.prow = sm.prow[cur ^ 1];
            hs_factor_panel<HS_FSB>(view, grp, n, k1, bw1, used, status_slot);
            LA_TOCK(7, 0);
        }
        {
            // every other strip of X and the strips of W, handed out dynamically: the update warps start at once, the
            // factor warps join when panel p+1 is factored
            const int nxs = nsx - (sn1 - sk0), tot = nxs + nsw;
            for (;;) {
                int s = 0;
                if ((tid & 31) == 0) s = atomicAdd(&sm.next, 1);
                s = __shfl_sync(0xffffffffu, s, 0);
                if (s >= tot) break;
                if (s < nsw) la_strip(panel, prow, W, ld, n, s * 8, nc, bw);
                else { const int sx = s - nsw; la_strip(panel, prow, X, ld, n, (sx < sk0 ? sx : sx + (sn1 - sk0)) * 8, n, bw); }
            }
            if (more) LA_TOCK(8, LA_U0); else { LA_TOCK(9, LA_U0); }
        }
        __syncthreads();
        if (more) { LA_TOCK(10, LA_U0); LA_TOCK(11, 0); }
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
    const HSAsm av = {&sm.panel[0][0], &sm.tab, sm.perm_prev, sm.pinv_prev};
    int n = 0;
    for (int hs = hs_begin; hs < hs_end; hs++) {
        const int i = hs >> 1, kind = hs & 1;
        cplx *Xp = kind ? X1 : X0, *Wp = kind ? W1 : W0, *Xn = kind ? X0 : X1, *Wn = kind ? W0 : W1;
        if (tid < HS_NMAX) { sm.perm_prev[tid] = sm.perm[tid]; sm.pinv_prev[tid] = sm.pinv[tid]; }
        __syncthreads();
        long long tc0 = a.prof ? clock64() : 0;
        hs_assemble<LA_NT, LA_RB, 1>(av, a, bl, i, kind, hs == 0, Xp, Wp, Xn, Wn);
        if (a.prof && tid == 0) sm.prof[0] += clock64() - tc0;
        n = half_count(M, kind == 0 ? ((i + 1) & 1) : (i & 1));
        la_gauss_jordan(sm, Xn, Wn, ld, n, nc, status_slot, a.prof ? a.prof + bl * 16 : nullptr, [&](int utid) {
            hs_assemble<LA_NT, LA_RB, 2>(av, a, bl, i, kind, hs == 0, Xp, Wp, Xn, Wn, utid, LA_NT - LA_NF);
        });
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
