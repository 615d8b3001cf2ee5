// half_sweep.cuh -- the fused sweep kernel of the half-slice formulation for M <= 256 (n = M/2 <= 128;
// the paper's 30 nm ribbon is M = 244, n = 122).
//
// One CTA owns one (device, energy) pair and runs its half-steps back to back (Eq. 4-5
// on the slicing B_0, F_0, B_1, F_1, ...; half_kernels.cuh states the recursion):
//     A = z - eps - C g_prev C^T  [- Sigma_L/R at the ends]         assembly, O(n^2)
//     [ g | P ] = A^-1 [ I | C P_prev ]                            ONE in-place Gauss-Jordan on the augmented matrix
// The propagator columns ride along as extra right-hand sides of the elimination, so inverse (8 n^3)
// and propagator product (8 n^3 real flops) are the same kernel loop: for every panel of 32 columns
//     1. the n x 32 panel is factored in shared memory with partial pivoting (rows never move; thread = row;
//        8-column sub-blocks in registers, the other panel columns by DMMA),
//     2. every other 8-column strip of [X | W] is updated in place, C += Mult * R on the FP64 tensor pipe
//        (mma.sync m8n8k4 = DMMA.8x8x4): a warp owns a strip, snapshots the strip's 32 pivot rows R in its B
//        fragments, reads Mult from the factored panel in shared memory and streams the C fragments L2 ->
//        registers -> L2 (no barrier and no shared-memory staging between the warps of an update).
// Rows are never exchanged: with p_k the pivot row of column k the result of an elimination sits at
//     (A^-1)[k][p_c] = X[p_k][c],   (A^-1 W)[k][:] = W[p_k][:]
// and the next half-step reads it through row / column maps (no unpermute pass).
// Assembly is mostly not a pass of its own:
//     kind B  A_B = z - eps - t^2 m' (.) gF_prev (.) m', W_B = t m' (.) PF_prev are the previous result scaled element by
//             element (+ a diagonal): left in place, in its permuted order, and transformed by whoever loads an element
//             first (panel 0 and its strips), HSXf;
//     kind F  A_F = z - eps - C gB C^T is a 2 x 2 stencil in rows and columns: gathered through shared memory
//             (hs_assemble); W_F = C PB is a two-row stencil, formed by the first panel's strips from the other buffer.
// State per matrix in HBM/L2: X (2 buffers), W (2 buffers), the two maps.  2 CTAs per SM (87 KB of shared memory each,
// 128 registers) so that one CTA's latency-bound pivot chain overlaps the other's DMMAs.
#pragma once
#include "half_kernels.cuh"
#include "rgf_common.cuh"

namespace rgf {

constexpr int HS_NT = 256, HS_NMAX = 128, HS_B = 32, HS_SB = 8;
constexpr int HS_LDP = HS_B + 4;        // 36: A-fragment reads of the panel conflict-free
constexpr int HS_LDR = HS_B + 2;        // 34: B-fragment reads conflict-free
constexpr int HS_RG = 2;                // row blocks of 8 per register tile of the strip update

struct HSweepArgs {
    int M, L, nh, ldn, n_E, bz0, nb;
    double eta, t;
    const double *energies, *onsite;
    const uint8_t *bond, *hop;
    const cplx *gL, *gR;
    cplx *X0, *X1, *P0, *P1;      // [nb][ldn*ldn] each
    int *perm;                    // [nb][2][HS_NMAX]: row and column maps of a matrix between launches
    int *status;                  // [nb]
    unsigned *pivmin;             // [nb] or NULL: min over all pivots of the top 24 bits of max(|re|, |im|)
    double *gsq;                  // [nb] (with pivmin): sum over the B half-steps of 1 / (smallest pivot)^2   (near-neutrality guard)
    int hs_begin, hs_end;         // half-steps [begin, end) of the whole sweep: hs = 2 i + kind
    int unit0, unit_len;          // this launch runs units unit0 + blockIdx.x; unit u = (matrix u % nb, half-steps
                                  // [hs_begin + (u / nb) unit_len, + unit_len)): rounds of units keep every CTA slot busy
    cplx *g_out, *P_out;          // after half-step hs_end - 1: g dense n x n (ld n) and P (ld nh), stride nh*nh; may be NULL
};

struct HSmem {
    cplx panel[HS_NMAX * HS_LDP];
    cplx Rs[HS_SB * HS_LDR];     // pivot rows of a sub-block (in-panel update)
    cplx crow[2 * (HS_NT / 32) * HS_SB];
    cplx cinv[2 * (HS_NT / 32)];
    alignas(16) unsigned ckey[2 * (HS_NT / 32)];
    int perm[HS_NMAX], pinv[HS_NMAX];                 // of the running elimination: pivot row of a column and its inverse
    int rmap[HS_NMAX], cmap[HS_NMAX];                 // logical row / column of the last result -> physical row / column
    int rmap_prev[HS_NMAX], cmap_prev[HS_NMAX];
    int prow[HS_B];
    unsigned pivmin;
    alignas(8) unsigned long long bar;                // mbarrier of the panel's TMA bulk copies
    // in-place assembly of a kind-B half-step (HSXf), per physical row / column of the previous result
    double xf_sr[HS_NMAX], xf_sw[HS_NMAX], xf_dre[HS_NMAX], xf_mc[HS_NMAX];
    short xf_dcol[HS_NMAX], xf_pa[HS_NMAX], xf_pb[HS_NMAX];
};

// per-row tables of the assembly; aliases HSmem::crow while no panel is being factored
struct HSTab {
    double eps[HS_NMAX];
    short ra[HS_NMAX], rb[HS_NMAX], ca[HS_NMAX], cb[HS_NMAX];
};
static_assert(sizeof(HSTab) <= sizeof(cplx) * 2 * (HS_NT / 32) * HS_SB, "HSTab must fit in HSmem::crow");

// named barrier over `nthreads` threads (whole warps)
__device__ __forceinline__ void hs_bar(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }

// The panel factorisation is written against a view of the shared-memory buffers and a description of the thread
// group that runs it (the whole CTA in the kernel below; a warp-specialised variant with four factor warps on one SM
// sub-partition and twelve update warps was measured 1.35x slower in round 1 and is not shipped: DESIGN.md section 9).
struct HSView {
    cplx *panel;          // [HS_NMAX][HS_LDP]
    cplx *Rs;             // [HS_SB][HS_LDR] snapshot of a sub-block's pivot rows
    cplx *crow, *cinv;    // candidate buffers [2][8][HS_SB], [2][8]
    unsigned *ckey;       // [2][8], 16-byte aligned
    int *prow, *perm, *pinv;
    unsigned *pivmin;
};
struct HSGroup {
    int r;                // row owned by this thread
    int slot, nslots;     // candidate slot of this warp, number of warps that search
    int gtid, gnt;        // thread index inside the group, group size
    int bar_pivot, n_pivot;   // barrier of the searching warps
    int bar_all;          // barrier of the whole group (gnt threads)
    int rbase;            // first of the 32 rows this warp updates in the in-panel DMMAs
    int nbsel, nbmod;     // ... for the column blocks whose running index % nbmod == nbsel
};

// One pivot step on column CC (static) of the thread's 8-column sub-block.  Candidate buffers alternate with
// the parity of CC, so one barrier per column suffices.  32-bit key = top 24 bits of |x|^2 (sign, exponent,
// 12 mantissa bits: any pivot within 2^-12 of the largest magnitude is as good as the maximum) and 255 - row,
// so the key is unique, names the row, and the lowest row wins ties.  The pivot row is not a divergent branch:
//   row[j] <- c + a * pivrow[j]   with (a, c) = (d, 0) on the pivot row and (-x d, row[j]) elsewhere, row[CC] <- a.
template <int CC, int SB>
__device__ __forceinline__ void hs_pivot_step(const HSView &sm, const HSGroup &gr, cplx (&row)[SB], bool &used, int kglob, int *status_slot)
{
    const int r = gr.r, warp = gr.slot, naw = gr.nslots;
    constexpr int NW = HS_NT / 32;
    constexpr int pb = (CC & 1) * NW;
    const cplx x = row[CC];
    // search key from max(|re|, |im|) (integer compare of the high words: no FP64 op on the critical path; the
    // chosen pivot is within sqrt(2) * (1 + 2^-12) of the largest modulus, as good for partial pivoting)
    const unsigned hre = (unsigned)__double2hiint(x.x) & 0x7fffffffu, him = (unsigned)__double2hiint(x.y) & 0x7fffffffu;
    const unsigned hi = used ? 0u : (max(hre, him) & 0xffffff00u);
    const unsigned key = hi | (unsigned)(255 - r);
    const double v = cabs2(x);                    // for the reciprocal; overlaps the warp reduction
    const unsigned wmax = __reduce_max_sync(0xffffffffu, key);
    if (key == wmax) {
        sm.ckey[pb + warp] = key;
        const double iv = hs_rcp(v);
        sm.cinv[pb + warp] = cmake(x.x * iv, -x.y * iv);
#pragma unroll
        for (int j = 0; j < SB; j++) if (j != CC) sm.crow[(pb + warp) * SB + j] = row[j];
    }
    hs_bar(gr.bar_pivot, gr.n_pivot);
    const uint4 k4 = *reinterpret_cast<const uint4 *>(&sm.ckey[pb]);
    unsigned best = k4.x;
    if (naw > 1) best = max(best, k4.y);
    if (naw > 2) best = max(best, k4.z);
    if (naw > 3) best = max(best, k4.w);
    if (naw > 4) {
        const uint4 k5 = *reinterpret_cast<const uint4 *>(&sm.ckey[pb + 4]);
        best = max(best, k5.x);
        if (naw > 5) best = max(best, k5.y);
        if (naw > 6) best = max(best, k5.z);
        if (naw > 7) best = max(best, k5.w);
    }
    const int pr = 255 - (int)(best & 0xffu), pw = pr >> 5;
    const cplx d = sm.cinv[pb + pw];
    const bool is_piv = (r == pr);
    const cplx nf = cmake(fma(-x.x, d.x, x.y * d.y), fma(-x.x, d.y, -x.y * d.x));     // -(x d)
    const cplx a = is_piv ? d : nf;
#pragma unroll
    for (int j = 0; j < SB; j++) {
        if (j == CC) { row[j] = a; continue; }
        const cplx pj = sm.crow[(pb + pw) * SB + j];
        cplx c = is_piv ? cmake(0.0, 0.0) : row[j];
        c.x = fma(a.x, pj.x, c.x); c.x = fma(-a.y, pj.y, c.x);
        c.y = fma(a.x, pj.y, c.y); c.y = fma(a.y, pj.x, c.y);
        row[j] = c;
    }
    if (is_piv) {
        if ((best >> 8) == 0u || best >= 0x7ff00000u) *status_slot = 1;
        atomicMin(sm.pivmin, best >> 8);
        used = true;
        sm.prow[kglob & (HS_B - 1)] = pr;
        sm.perm[kglob] = pr;
        sm.pinv[pr] = kglob;
    }
}

// in-panel update behind sub-block s (columns [c0, c0 + ncols) of the panel, pivot rows snapshotted in sm.Rs):
// panel[:, J] += (N'_s - E_s) (n x SB) * Rs (SB x |J|) on DMMA; a warp takes the 32 rows from gr.rbase and the column blocks
// whose running index % gr.nbmod == gr.nbsel
template <int SB>
__device__ __forceinline__ void hs_inpanel_update(const HSView &sm, const HSGroup &gr, int n, int bw, int s, int c0, int ncols)
{
    constexpr int LDP = HS_LDP, LDR = HS_LDR;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    cplx *panel = sm.panel;
    const cplx *Rs = sm.Rs;
    const int nbmax = (bw + 7) / 8;
    // other panel columns: panel[:, J] += (N'_s - E_s) (n x 8) * Rs (8 x |J|) on DMMA; a warp takes 32 rows
    // and the column blocks whose running index % nbmod == nbsel
    const int rbase = gr.rbase;
    if (rbase < n) {
        constexpr int KQ = SB / 4;
        int pk[KQ];
#pragma unroll
        for (int q = 0; q < KQ; q++) pk[q] = (q * 4 + t < ncols) ? sm.prow[c0 + q * 4 + t] : -1;
        cplx a[KQ][4];
#pragma unroll
        for (int q = 0; q < KQ; q++)
#pragma unroll
            for (int i = 0; i < 4; i++) {
                const int rr = rbase + i * 8 + g;
                a[q][i] = panel[rr * LDP + c0 + q * 4 + t];
                if (rr == pk[q]) a[q][i].x -= 1.0;
            }
        int cnt = 0;
        for (int nb = 0; nb < nbmax; nb++) {
            if (SB == 8 && nb == s) continue;
            if (((cnt++) % gr.nbmod) != gr.nbsel) continue;
            double cre[4][2], cim[4][2];
            cplx *Cw = panel + rbase * LDP + nb * 8;
#pragma unroll
            for (int i = 0; i < 4; i++) {
                const cplx v0 = Cw[(i * 8 + g) * LDP + 2 * t], v1 = Cw[(i * 8 + g) * LDP + 2 * t + 1];
                cre[i][0] = v0.x; cim[i][0] = v0.y; cre[i][1] = v1.x; cim[i][1] = v1.y;
            }
#pragma unroll
            for (int q = 0; q < KQ; q++) {
                const cplx bb = Rs[(q * 4 + t) * LDR + nb * 8 + g];
#pragma unroll
                for (int i = 0; i < 4; i++) zmma884(cre[i], cim[i], a[q][i].x, a[q][i].y, -a[q][i].y, bb.x, bb.y);
            }
#pragma unroll
            for (int i = 0; i < 4; i++) {
                Cw[(i * 8 + g) * LDP + 2 * t] = cmake(cre[i][0], cim[i][0]);
                Cw[(i * 8 + g) * LDP + 2 * t + 1] = cmake(cre[i][1], cim[i][1]);
            }
        }
    }
}

// ---- panel factorisation in shared memory: columns [k0, k0 + bw) of all n rows --------------------
// On entry sm.panel[r][c] = X[r][k0 + c] (zero for c >= bw, r >= n).  On exit sm.panel = N' (the
// transformed columns), sm.prow[c] = pivot row of column k0 + c, perm / pinv updated, used |= pivot.
// SB = columns per register sub-block: 8 (two DMMA k-steps per in-panel update) or 4 (one k-step; half the FP64
// instructions per pivot step, which is what counts when the pivot chain runs beside another warp's DMMAs)
template <int SB = HS_SB>
__device__ __forceinline__ void hs_factor_panel(const HSView &sm, const HSGroup &gr, int n, int k0, int bw, bool &used, int *status_slot)
{
    constexpr int B = HS_B, LDP = HS_LDP, LDR = HS_LDR;
    static_assert(SB == 8 || SB == 4, "sub-block width");
    const int r = gr.r;
    const bool has_row = r < n;
    cplx *panel = sm.panel;
    cplx *Rs = sm.Rs;
    for (int s = 0; s < B / SB; s++) {
        const int c0 = s * SB;
        const int ncols = bw - c0 < SB ? bw - c0 : SB;
        if (ncols <= 0) break;
        cplx row[SB];
        if (has_row) {
#pragma unroll
            for (int j = 0; j < SB; j++) row[j] = panel[r * LDP + c0 + j];
        } else {
#pragma unroll
            for (int j = 0; j < SB; j++) row[j] = cmake(0.0, 0.0);
        }
        if (gr.slot < gr.nslots) {
            const int kg = k0 + c0;
            hs_pivot_step<0, SB>(sm, gr, row, used, kg, status_slot);
            if (ncols > 1) hs_pivot_step<1, SB>(sm, gr, row, used, kg + 1, status_slot);
            if (ncols > 2) hs_pivot_step<2, SB>(sm, gr, row, used, kg + 2, status_slot);
            if (ncols > 3) hs_pivot_step<3, SB>(sm, gr, row, used, kg + 3, status_slot);
            if constexpr (SB == 8) {
                if (ncols > 4) hs_pivot_step<4, SB>(sm, gr, row, used, kg + 4, status_slot);
                if (ncols > 5) hs_pivot_step<5, SB>(sm, gr, row, used, kg + 5, status_slot);
                if (ncols > 6) hs_pivot_step<6, SB>(sm, gr, row, used, kg + 6, status_slot);
                if (ncols > 7) hs_pivot_step<7, SB>(sm, gr, row, used, kg + 7, status_slot);
            }
        }
        hs_bar(gr.bar_all, gr.gnt);
        if (has_row) {
#pragma unroll
            for (int j = 0; j < SB; j++) panel[r * LDP + c0 + j] = row[j];
        }
        if (bw > SB) {
            // snapshot of the sub-block's pivot rows; zero in the sub-block's own columns (for SB = 4 they share a DMMA
            // column block with four columns that are updated)
            for (int e = gr.gtid; e < SB * B; e += gr.gnt) {
                const int k = e / B, c = e % B;
                const bool own = c >= c0 && c < c0 + SB;
                Rs[k * LDR + c] = (k < ncols && !own) ? panel[sm.prow[c0 + k] * LDP + c] : cmake(0.0, 0.0);
            }
            hs_bar(gr.bar_all, gr.gnt);
            hs_inpanel_update<SB>(sm, gr, n, bw, s, c0, ncols);
            hs_bar(gr.bar_all, gr.gnt);
        }
    }
}

// view / group of the whole-CTA kernel: thread = row, all eight warps in the in-panel DMMAs
__device__ __forceinline__ HSView hs_view(HSmem &sm)
{
    HSView v;
    v.panel = sm.panel; v.Rs = sm.Rs; v.crow = sm.crow; v.cinv = sm.cinv; v.ckey = sm.ckey;
    v.prow = sm.prow; v.perm = sm.perm; v.pinv = sm.pinv; v.pivmin = &sm.pivmin;
    return v;
}
__device__ __forceinline__ HSGroup hs_group_cta(int n)
{
    HSGroup g;
    const int tid = threadIdx.x, warp = tid >> 5;
    g.r = tid; g.slot = warp; g.nslots = (n + 31) >> 5; g.gtid = tid; g.gnt = HS_NT;
    g.bar_pivot = 1; g.n_pivot = g.nslots * 32; g.bar_all = 0;
    g.rbase = (warp & 3) * 32; g.nbsel = warp >> 2; g.nbmod = 2;
    return g;
}

// ---- in-place assembly of a kind-B half-step, applied to an element while it is loaded ---------------------------
// A_B = z - eps_B - t^2 m' (.) gF_prev (.) m' and W_B = t m' (.) PF_prev are the previous result scaled element by
// element plus a diagonal (half_kernels.cuh): nothing moves, so the previous result is left where it is (rows and
// columns in the permuted order the elimination produced) and turned into [A | W] on the fly by whoever loads an
// element first -- the load of panel 0 and the strips of its update touch every element exactly once.  Tables are per
// PHYSICAL row rho / column gamma of the previous result:  x' = sr[rho] mc[gamma] x  (+ (dre[rho], eta) at gamma =
// dcol[rho], the position of the atom's own diagonal element),  w' = sw[rho] w.
struct HSXf {
    const double *sr, *sw, *dre, *mc;
    const short *dcol;
    double eta;
    // kind-F half-steps: W = C P_prev is a two-row stencil of the previous propagator (other buffer), W[r] = t (Wp[pa[r]] +
    // Wp[pb[r]]), pa / pb = physical rows of the lower / upper B neighbour or -1; also formed by whoever loads first
    const cplx *Wp;
    const short *pa, *pb;
    double t;
};
// TF: 0 = plain load, 1 = element of X (kind B), 2 = element of W (kind B), 3 = W of a kind-F half-step (hs_wf_load)
template <int TF>
__device__ __forceinline__ cplx hs_xf(const HSXf &xf, cplx v, int rho, int gamma)
{
    if (TF == 1) {
        const double sc = xf.sr[rho] * xf.mc[gamma];
        v.x *= sc; v.y *= sc;
        if (gamma == xf.dcol[rho]) { v.x += xf.dre[rho]; v.y += xf.eta; }
    } else if (TF == 2) {
        const double sc = xf.sw[rho];
        v.x *= sc; v.y *= sc;
    }
    return v;
}

// two adjacent elements (row r, columns gamma0, gamma0 + 1; gamma0 even) of W = C P_prev
__device__ __forceinline__ void hs_wf_load2(const HSXf &xf, int ld, int r, int gamma0, double &a0, double &a1, double &a2, double &a3)
{
    const int pa = xf.pa[r], pb = xf.pb[r];
    double b0 = 0.0, b1 = 0.0, b2 = 0.0, b3 = 0.0, c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0;
    if (pa >= 0) ld256cg(xf.Wp + (long long)pa * ld + gamma0, b0, b1, b2, b3);
    if (pb >= 0) ld256cg(xf.Wp + (long long)pb * ld + gamma0, c0, c1, c2, c3);
    a0 = xf.t * (b0 + c0); a1 = xf.t * (b1 + c1); a2 = xf.t * (b2 + c2); a3 = xf.t * (b3 + c3);
}
__device__ __forceinline__ cplx hs_wf_load1(const HSXf &xf, int ld, int r, int gamma)
{
    const int pa = xf.pa[r], pb = xf.pb[r];
    cplx va = cmake(0.0, 0.0), vb = cmake(0.0, 0.0);
    if (pa >= 0) va = ldcg(xf.Wp + (long long)pa * ld + gamma);
    if (pb >= 0) vb = ldcg(xf.Wp + (long long)pb * ld + gamma);
    return cmake(xf.t * (va.x + vb.x), xf.t * (va.y + vb.y));
}

// ---- barrier-free update of one 8-column strip: C[:, col0 .. col0+8) += Mult (n x 32, sm.panel) * R ---------------
// R = the strip's 32 pivot rows, snapshotted into the warp's B fragments (registers) before any row of the strip is
// written, so a warp needs nothing from the other warps: no R staging through shared memory, no barrier per chunk, and
// the warps drift apart so that one warp's loads / stores overlap another's DMMAs.  Row groups of 8 RG rows; the next
// group's C fragments are in flight from L2 while the current group is on the tensor pipe.
template <int RG>
struct HSAcc { double re[RG][2], im[RG][2]; };

template <int RG, int TF>
__device__ __forceinline__ void hs_acc_load(HSAcc<RG> &h, const cplx *Cl, int ld, int n, int r0, bool cok, const HSXf &xf, int gamma0)
{
    const int lane = threadIdx.x & 31, g = lane >> 2;
#pragma unroll
    for (int i = 0; i < RG; i++) {
        const int rr = r0 + i * 8 + g;
        double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
        if (rr < n && cok) {
            // elements (rr, c) and (rr, c + 1), c even: one 32-byte sector, one LDG.256.  c + 1 may be the padding column.
            if (TF == 3) hs_wf_load2(xf, ld, rr, gamma0, a0, a1, a2, a3);
            else ld256cg(Cl + (long long)rr * ld, a0, a1, a2, a3);
            if (TF == 1 || TF == 2) {
                const cplx v0 = hs_xf<TF>(xf, cmake(a0, a1), rr, gamma0), v1 = hs_xf<TF>(xf, cmake(a2, a3), rr, gamma0 + 1);
                a0 = v0.x; a1 = v0.y; a2 = v1.x; a3 = v1.y;
            }
        }
        h.re[i][0] = a0; h.im[i][0] = a1; h.re[i][1] = a2; h.im[i][1] = a3;
    }
}
template <int RG>
__device__ __forceinline__ void hs_acc_store(const HSAcc<RG> &h, cplx *Cl, int ld, int n, int r0, bool cok)
{
    const int lane = threadIdx.x & 31, g = lane >> 2;
#pragma unroll
    for (int i = 0; i < RG; i++) {
        const int rr = r0 + i * 8 + g;
        if (rr < n && cok) st256(Cl + (long long)rr * ld, h.re[i][0], h.im[i][0], h.re[i][1], h.im[i][1]);
    }
}
// FULL = number of k-steps of 4 in straight-line code (8: a full 32-column panel; 7: a panel of 25 .. 28 columns, the last one of
// n = 122 is 26 wide), 0 = generic loop over kq steps
template <int RG, int FULL>
__device__ __forceinline__ void hs_acc_compute(HSAcc<RG> &h, const cplx *panel, int r0, const cplx (&bb)[8], int kq)
{
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const cplx *cA = panel + (r0 + g) * HS_LDP + t;
    if (FULL > 0) {
        // straight-line code: the A fragments of step q + 1 are loaded before the DMMAs of step q
        cplx a[2][RG];
#pragma unroll
        for (int i = 0; i < RG; i++) a[0][i] = cA[i * 8 * HS_LDP];
#pragma unroll
        for (int q = 0; q < FULL; q++) {
            if (q + 1 < FULL) {
#pragma unroll
                for (int i = 0; i < RG; i++) a[(q + 1) & 1][i] = cA[i * 8 * HS_LDP + (q + 1) * 4];
            }
#pragma unroll
            for (int i = 0; i < RG; i++) zmma884(h.re[i], h.im[i], a[q & 1][i].x, a[q & 1][i].y, -a[q & 1][i].y, bb[q].x, bb[q].y);
        }
    } else {
#pragma unroll
        for (int q = 0; q < 8; q++) {
            if (q < kq) {
                cplx a[RG];
#pragma unroll
                for (int i = 0; i < RG; i++) a[i] = cA[i * 8 * HS_LDP + q * 4];
#pragma unroll
                for (int i = 0; i < RG; i++) zmma884(h.re[i], h.im[i], a[i].x, a[i].y, -a[i].y, bb[q].x, bb[q].y);
            }
        }
    }
}

// Mult columns / R rows beyond the panel width are zero, so a narrow last panel only skips DMMAs (FULL = false).
template <int RG, int FULL, int TF>
__device__ __forceinline__ void hs_strip_update(const cplx *panel, const int *prow, cplx *Cg, int ld, int n, int col0, int ncols, int bw,
                                                const HSXf &xf)
{
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    // B fragments: the strip's (<= 32) pivot rows, read from L2 before any row of the strip is written
    cplx bb[8];
    {
        const bool colok = col0 + g < ncols;
#pragma unroll
        for (int q = 0; q < 8; q++) {
            const int k = q * 4 + t;
            bb[q] = cmake(0.0, 0.0);
            if (k < bw && colok) {
                const int rho = prow[k];
                if (TF == 3) bb[q] = hs_wf_load1(xf, ld, rho, col0 + g);
                else bb[q] = hs_xf<TF>(xf, ldcg(Cg + (long long)rho * ld + col0 + g), rho, col0 + g);
            }
        }
    }
    const int kq = (bw + 3) >> 2;
    const int gamma0 = col0 + 2 * t;
    const bool cok = gamma0 < ncols;
    cplx *Cl = Cg + gamma0;
    constexpr int GR = 8 * RG;
    HSAcc<RG> h0, h1;
    hs_acc_load<RG, TF>(h0, Cl, ld, n, 0, cok, xf, gamma0);
    for (int r0 = 0; r0 < n; r0 += 2 * GR) {
        hs_acc_load<RG, TF>(h1, Cl, ld, n, r0 + GR, cok, xf, gamma0);
        hs_acc_compute<RG, FULL>(h0, panel, r0, bb, kq);
        hs_acc_store<RG>(h0, Cl, ld, n, r0, cok);
        hs_acc_load<RG, TF>(h0, Cl, ld, n, r0 + 2 * GR, cok, xf, gamma0);
        if (r0 + GR < n) {
            hs_acc_compute<RG, FULL>(h1, panel, r0 + GR, bb, kq);
            hs_acc_store<RG>(h1, Cl, ld, n, r0 + GR, cok);
        }
    }
}

// ---- [X | W] <- A^-1 [I | W] in place; fills sm.perm / sm.pinv.  X holds A on entry (xtf = 0) or the previous result
// that HSXf turns into A while panel 0 is loaded and applied (xtf = 1); W likewise: wtf = 0 (W in place), 2 (previous
// propagator, scaled in place) or 3 (stencil of the previous propagator in the other buffer) ---------------------------------------
__device__ __forceinline__ void hs_gauss_jordan(HSmem &sm, cplx *X, cplx *W, int ld, int n, int nc, int *status_slot,
                                                int xtf, int wtf, const HSXf &xf, unsigned &tma_phase)
{
    const int tid = threadIdx.x;
    bool used = !(tid < n);
    const HSView view = hs_view(sm);
    const HSGroup grp = hs_group_cta(n);
    const int nsx = (n + 7) >> 3, nsw = (nc + 7) >> 3;
    for (int k0 = 0; k0 < n; k0 += HS_B) {
        const int bw = (n - k0 < HS_B) ? (n - k0) : HS_B;
        const bool tf = (xtf | wtf) != 0 && k0 == 0;
        if (!(tf && xtf)) {
            // the n x bw panel by TMA: one bulk copy per row (bw contiguous elements of X), all completing on one mbarrier;
            // the padding (rows >= n, columns >= bw) is zeroed with plain stores, which touch none of the copied bytes
            if (tid == 0) tma_expect(&sm.bar, (unsigned)(n * bw) * (unsigned)sizeof(cplx));
            if (tid < n) {
                tma_fence_proxy();          // this buffer was last written / read through the generic proxy
                tma_load_row(sm.panel + tid * HS_LDP, X + (long long)tid * ld + k0, (unsigned)bw * (unsigned)sizeof(cplx), &sm.bar);
                for (int c = bw; c < HS_B; c++) sm.panel[tid * HS_LDP + c] = cmake(0.0, 0.0);
            } else if (tid < HS_NMAX) {
                for (int c = 0; c < HS_B; c++) sm.panel[tid * HS_LDP + c] = cmake(0.0, 0.0);
            }
            tma_wait(&sm.bar, tma_phase);
            tma_phase ^= 1u;
        } else {
            // panel 0 of an in-place half-step: transformed on its way to shared memory, 8 loads in flight per thread
            constexpr int PER = 8;
            for (int e0 = 0; e0 < HS_NMAX * HS_B; e0 += PER * HS_NT) {
                cplx v[PER];
#pragma unroll
                for (int k = 0; k < PER; k++) {
                    const int e = e0 + k * HS_NT + tid, rr = e / HS_B, c = e % HS_B;
                    v[k] = cmake(0.0, 0.0);
                    if (rr < n && c < bw) v[k] = ldcg(X + (long long)rr * ld + c);
                }
#pragma unroll
                for (int k = 0; k < PER; k++) {
                    const int e = e0 + k * HS_NT + tid, rr = e / HS_B, c = e % HS_B;
                    if (rr < n && c < bw) v[k] = hs_xf<1>(xf, v[k], rr, c);
                    sm.panel[rr * HS_LDP + c] = v[k];
                }
            }
        }
        __syncthreads();
        hs_factor_panel<HS_SB>(view, grp, n, k0, bw, used, status_slot);
        // N' -> X[:, K];  then the panel becomes Mult = N' - E (E[prow[c]][c] = 1)
        for (int e = tid; e < n * HS_B; e += HS_NT) {
            const int rr = e / HS_B, c = e % HS_B;
            if (c < bw) X[(long long)rr * ld + k0 + c] = sm.panel[rr * HS_LDP + c];
        }
        __syncthreads();
        if (tid < bw) sm.panel[sm.prow[tid] * HS_LDP + tid].x -= 1.0;
        __syncthreads();
        // strip list: the 8-column strips of X except the panel's own four, then the strips of W; warp w takes
        // strips w, w + 8, ...
        const int sk0 = k0 >> 3;
        const int sk1 = (sk0 + HS_B / 8 < nsx) ? sk0 + HS_B / 8 : nsx;
        const int nxs = nsx - (sk1 - sk0), tot = nxs + nsw;
        auto strip_of = [&](int s, cplx *&Cg, int &col0, int &ncols) {
            const bool isx = s < nxs;
            Cg = isx ? X : W;
            col0 = (isx ? (s < sk0 ? s : s + (sk1 - sk0)) : s - nxs) * 8; ncols = isx ? n : nc;
            return isx;
        };
        for (int s = tid >> 5; s < tot; s += HS_NT / 32) {
            cplx *Cg; int col0, ncols;
            const bool isx = strip_of(s, Cg, col0, ncols);
            const int tfs = tf ? (isx ? xtf : wtf) : 0;
            // straight-line code over 8 k-steps (bw > 28) or 7 (24 < bw <= 28: the last panel of n = 122 is 26 wide); Mult columns /
            // pivot rows beyond the panel width are zero, so a k-step that is only partly filled just adds DMMAs on zeros
            const int full = bw > 28 ? 8 : (bw > 24 ? 7 : 0);
#define HS_STRIP(F, T) hs_strip_update<HS_RG, F, T>(sm.panel, sm.prow, Cg, ld, n, col0, ncols, bw, xf)
            if (full == 8) {
                if (tfs == 0) HS_STRIP(8, 0); else if (tfs == 1) HS_STRIP(8, 1); else if (tfs == 2) HS_STRIP(8, 2); else HS_STRIP(8, 3);
            } else if (full == 7 && tfs == 0) {
                HS_STRIP(7, 0);
            } else {
                if (tfs == 0) HS_STRIP(0, 0); else if (tfs == 1) HS_STRIP(0, 1); else if (tfs == 2) HS_STRIP(0, 2); else HS_STRIP(0, 3);
            }
#undef HS_STRIP
        }
        __syncthreads();
    }
}

// ---- assembly of A (into Xn) and of W = C P_prev (into Wn) for half-step (i, kind) -------------------------
// g_prev[k][m] = Xp[rmap[k]][cmap[m]], P_prev[k][:] = Wp[rmap[k]][:]; blocks of 16 output rows,
// the physical rows they need staged in the (idle) panel buffer so that every L2 read is a full row.
struct HSAsm {
    cplx *stage;                       // staging area of 2 (RB + 2) rows of HS_NMAX elements (the idle panel buffer)
    HSTab *tb;                         // per-row tables (alias the idle candidate buffers)
    const int *rmap, *cmap;            // logical row / column of the previous result -> physical row / column
};
// PART 0: A and W by all NT threads; 1: the tables and A only (all NT threads; ends with a barrier); 2: W only, by the
// wnt threads wtid = 0 .. wnt-1 (no barrier; needs the tables of PART 1)
template <int NT, int RB, int PART = 0>
__device__ __forceinline__ void hs_assemble(const HSAsm &sm, const HSweepArgs &a, int bl, int i, int kind, bool first,
                                            const cplx *Xp, const cplx *Wp, cplx *Xn, cplx *Wn, int wtid = threadIdx.x, int wnt = NT)
{
    constexpr int HS_NT = NT;        // threads that run the assembly (the whole CTA of either kernel)
    const int tid = threadIdx.x, M = a.M, L = a.L, ld = a.ldn, nc = M / 2;
    const int bz = a.bz0 + bl, d = bz / a.n_E, e = bz % a.n_E;
    const double t2 = a.t * a.t, E = a.energies[e];
    const double *eps = a.onsite + ((long long)d * L + i) * M;
    const long long MM = (long long)M * M;
    const int par = kind == 0 ? ((i + 1) & 1) : (i & 1);
    const int n = half_count(M, par), nprev = kind == 0 ? n : half_count(M, 1 - par);
    const uint8_t *mk = a.bond + ((long long)d * (L + 1) + i) * M;        // m'_{i-1}
    const uint8_t *mr = a.bond + ((long long)d * (L + 1) + L) * M;        // m'_{L-1}
    const uint8_t *hp = a.hop + ((long long)d * L + i) * M;
    cplx *stage = sm.stage;
    if (first) {
        // half-step 0 (B_0): g_prev = surface Green's function of the left lead (slice -1, same atoms j), W = I
        const cplx *gl = a.gL + (long long)e * MM;
        if (PART != 2)
        for (int idx = tid; idx < n * n; idx += HS_NT) {
            const int r = idx / n, c = idx % n, jr = 2 * r + par, jc = 2 * c + par;
            cplx v = cmake(0.0, 0.0);
            if (r == c) v = cmake(E - eps[jr], a.eta);
            if (mk[jr] && mk[jc]) { const cplx g = gl[(long long)jr * M + jc]; v.x -= t2 * g.x; v.y -= t2 * g.y; }
            Xn[(long long)r * ld + c] = v;
        }
        if (PART != 1)
        for (int idx = wtid; idx < n * nc; idx += wnt) {
            const int r = idx / nc, c = idx % nc;
            Wn[(long long)r * ld + c] = cmake(r == c ? 1.0 : 0.0, 0.0);
        }
        if (PART == 1) __syncthreads();
        return;
    }
    const cplx *gr = a.gR + (long long)e * MM;
    const bool last = (kind == 1 && i == L - 1);
    // per-row tables of this half-step (the candidate buffers of the pivot search are idle here):
    //   kind B: ra[r] = m'[r];                       ca[c] = m'[c] ? physical column of g_prev[.][c] : -1
    //   kind F: ra/rb[r] = lower / upper B neighbour; ca/cb[c] = physical column of that neighbour, or -1
    HSTab &tb = *sm.tb;
    if (PART != 2) {
    if (tid < n) {
        const int r = tid;
        tb.eps[r] = E - eps[2 * r + par];
        if (kind == 0) {
            const int m = mk[2 * r + par] ? 1 : 0;
            tb.ra[r] = (short)m; tb.rb[r] = -1;
            tb.ca[r] = (short)(m ? sm.cmap[r] : -1); tb.cb[r] = -1;
        } else {
            const int s0 = half_nbr(r, par, 0, M, hp), s1 = half_nbr(r, par, 1, M, hp);
            tb.ra[r] = (short)s0; tb.rb[r] = (short)s1;
            tb.ca[r] = (short)(s0 >= 0 ? sm.cmap[s0] : -1);
            tb.cb[r] = (short)(s1 >= 0 ? sm.cmap[s1] : -1);
        }
    }
    __syncthreads();
    // blocks of 16 output rows; the (<= 18) physical rows a block needs are staged by cp.async into one of two areas of
    // the panel buffer, the next block's rows in flight while this block is computed
    constexpr int AREA = (RB + 2) * HS_NMAX;
    auto rows_of = [&](int r0, int &slo, int &nst) {
        const int r1 = (r0 + RB < n) ? r0 + RB : n;
        int shi = r1 - 1;
        slo = r0;
        if (kind == 1) { if (par == 0) slo = r0 - 1; else shi = r1; }
        if (slo < 0) slo = 0;
        if (shi > nprev - 1) shi = nprev - 1;
        nst = shi - slo + 1;
    };
    auto stage_rows = [&](int r0, int area) {
        int slo, nst;
        rows_of(r0, slo, nst);
        cplx *dst = stage + area * AREA;
        // thread = (row tid / 128 + k NT / 128, column tid % 128): no division by the runtime ld
        const int c = tid & (HS_NMAX - 1);
        if (c < ld)
            for (int sl = tid / HS_NMAX; sl < nst; sl += HS_NT / HS_NMAX)
                cp_async16(dst + sl * HS_NMAX + c, Xp + (long long)sm.rmap[slo + sl] * ld + c, 16);
        cp_async_commit();
    };
    stage_rows(0, 0);
    for (int r0 = 0, blk = 0; r0 < n; r0 += RB, blk++) {
        const int r1 = (r0 + RB < n) ? r0 + RB : n;
        int slo, nst;
        rows_of(r0, slo, nst);
        if (r0 + RB < n) { stage_rows(r0 + RB, (blk + 1) & 1); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncthreads();
        const cplx *st = stage + (blk & 1) * AREA;
        const int c = tid & (HS_NMAX - 1);
        const int ca = c < n ? tb.ca[c] : -1, cb = c < n ? tb.cb[c] : -1;
        if (c < n)
        for (int r = r0 + tid / HS_NMAX; r < r1; r += HS_NT / HS_NMAX) {
            cplx v = cmake(0.0, 0.0);
            if (r == c) v = cmake(tb.eps[r], a.eta);
            double sx = 0.0, sy = 0.0;
            if (kind == 0) {
                if (tb.ra[r] && ca >= 0) { const cplx g = st[(r - slo) * HS_NMAX + ca]; sx = g.x; sy = g.y; }
            } else {
                const int ua = tb.ra[r], ub = tb.rb[r];
                if (ua >= 0) {
                    const cplx *sr = st + (ua - slo) * HS_NMAX;
                    if (ca >= 0) { const cplx g = sr[ca]; sx += g.x; sy += g.y; }
                    if (cb >= 0) { const cplx g = sr[cb]; sx += g.x; sy += g.y; }
                }
                if (ub >= 0) {
                    const cplx *sr = st + (ub - slo) * HS_NMAX;
                    if (ca >= 0) { const cplx g = sr[ca]; sx += g.x; sy += g.y; }
                    if (cb >= 0) { const cplx g = sr[cb]; sx += g.x; sy += g.y; }
                }
            }
            v.x -= t2 * sx; v.y -= t2 * sy;
            if (last) {
                const int jr = 2 * r + par, jc = 2 * c + par;
                if (mr[jr] && mr[jc]) { const cplx g = gr[(long long)jr * M + jc]; v.x -= t2 * g.x; v.y -= t2 * g.y; }
            }
            Xn[(long long)r * ld + c] = v;
        }
        __syncthreads();
    }
    }
    if (PART == 1) return;
    // W = C P_prev: coalesced rows straight from L2, 6 independent elements per thread in flight
    const int nel = n * nc;
    constexpr int WB = 6;
    for (int base = 0; base < nel; base += WB * wnt) {
        cplx va[WB], vb[WB];
        int rr[WB], cc[WB];
#pragma unroll
        for (int k = 0; k < WB; k++) {
            const int idx = base + k * wnt + wtid;
            va[k] = cmake(0.0, 0.0); vb[k] = cmake(0.0, 0.0);
            rr[k] = -1;
            if (idx < nel) {
                const int r = idx / nc, c = idx - r * nc;
                rr[k] = r; cc[k] = c;
                if (kind == 0) {
                    if (tb.ra[r]) va[k] = ldcg(Wp + (long long)sm.rmap[r] * ld + c);
                } else {
                    const int ua = tb.ra[r], ub = tb.rb[r];
                    if (ua >= 0) va[k] = ldcg(Wp + (long long)sm.rmap[ua] * ld + c);
                    if (ub >= 0) vb[k] = ldcg(Wp + (long long)sm.rmap[ub] * ld + c);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < WB; k++)
            if (rr[k] >= 0) Wn[(long long)rr[k] * ld + cc[k]] = cmake(a.t * (va[k].x + vb[k].x), a.t * (va[k].y + vb[k].y));
    }
    if (PART == 0) __syncthreads();          // the tables alias the pivot-search buffers
}

// buffer (0 / 1) that half-step hs leaves its result in: half-step 0 (B_0, assembled from the lead) writes buffer 1, every
// F half-step reads one buffer and writes the other, every later B half-step works in place
__device__ __forceinline__ int hs_out_buf(int hs) { return (((hs + 1) >> 1) & 1) ^ 1; }

// ---- the sweep: one CTA per matrix, half-steps [hs_begin, hs_end) ----------------------------------------
__global__ void __launch_bounds__(HS_NT, 2) half_sweep_kernel(HSweepArgs a)
{
    extern __shared__ __align__(16) unsigned char hs_smem_raw[];
    HSmem &sm = *reinterpret_cast<HSmem *>(hs_smem_raw);
    const int tid = threadIdx.x, M = a.M, L = a.L, ld = a.ldn, nc = M / 2;
    const long long unit = (long long)a.unit0 + blockIdx.x;
    const int bl = (int)(unit % a.nb);
    const int hs_begin = a.hs_begin + (int)(unit / a.nb) * a.unit_len;
    const int hs_end = (hs_begin + a.unit_len < a.hs_end) ? hs_begin + a.unit_len : a.hs_end;
    if (hs_begin >= hs_end) return;
    const long long xs = (long long)ld * ld;
    cplx *const X0 = a.X0 + bl * xs, *const X1 = a.X1 + bl * xs, *const W0 = a.P0 + bl * xs, *const W1 = a.P1 + bl * xs;
    int *gmaps = a.perm + (long long)bl * 2 * HS_NMAX;
    int *status_slot = a.status + bl;
    unsigned kmin = 0xffffffffu;          // thread 0: smallest pivot key of the unit, and the guard's sum
    unsigned tma_phase = 0u;
    if (tid == 0) tma_bar_init(&sm.bar, 1);
    double gsq = 0.0;
    if (hs_begin > 0) {
        if (tid < HS_NMAX) { sm.rmap[tid] = gmaps[tid]; sm.cmap[tid] = gmaps[HS_NMAX + tid]; }
        __syncthreads();
    }
    const int bz = a.bz0 + bl, dev = bz / a.n_E;
    const double E = a.energies[bz % a.n_E];
    HSXf xf = {sm.xf_sr, sm.xf_sw, sm.xf_dre, sm.xf_mc, sm.xf_dcol, a.eta, nullptr, sm.xf_pa, sm.xf_pb, a.t};
    int n = 0;
    for (int hs = hs_begin; hs < hs_end; hs++) {
        const int i = hs >> 1, kind = hs & 1;
        const int ob = hs_out_buf(hs), ib = hs > 0 ? hs_out_buf(hs - 1) : 0;
        cplx *Xn = ob ? X1 : X0, *Wn = ob ? W1 : W0;
        const cplx *Xp = ib ? X1 : X0, *Wp = ib ? W1 : W0;
        const bool inplace = kind == 0 && hs > 0;
        const int par = kind == 0 ? ((i + 1) & 1) : (i & 1);
        n = half_count(M, par);
        if (tid < HS_NMAX) { sm.rmap_prev[tid] = sm.rmap[tid]; sm.cmap_prev[tid] = sm.cmap[tid]; }
        if (tid == 0) sm.pivmin = 0xffffffffu;
        __syncthreads();
        if (inplace) {
            // tables of the in-place assembly (HSXf): atom r of this B half sits in physical row rmap[r] and its column
            // in physical column cmap[r] of the previous (F) result
            if (tid < n) {
                const int r = tid, j = 2 * r + par, rho = sm.rmap_prev[r], gam = sm.cmap_prev[r];
                const double m = a.bond[((long long)dev * (L + 1) + i) * M + j] ? 1.0 : 0.0;      // m'_{i-1}
                sm.xf_sr[rho] = -a.t * a.t * m; sm.xf_sw[rho] = a.t * m;
                sm.xf_dre[rho] = E - a.onsite[((long long)dev * L + i) * M + j];
                sm.xf_dcol[rho] = (short)gam;
                sm.xf_mc[gam] = m;
            }
        } else {
            static_assert(2 * (16 + 2) * HS_NMAX <= HS_NMAX * HS_LDP, "two staging areas must fit in the panel buffer");
            const HSAsm av = {sm.panel, reinterpret_cast<HSTab *>(sm.crow), sm.rmap_prev, sm.cmap_prev};
            if (hs == 0) hs_assemble<HS_NT, 16, 0>(av, a, bl, i, kind, true, Xp, Wp, Xn, Wn);
            else {
                // kind F: A is gathered through shared memory; W = C P_prev is left to the first panel's strips
                if (tid < n) {
                    const uint8_t *hp = a.hop + ((long long)dev * L + i) * M;
                    const int s0 = half_nbr(tid, par, 0, M, hp), s1 = half_nbr(tid, par, 1, M, hp);
                    sm.xf_pa[tid] = (short)(s0 >= 0 ? sm.rmap_prev[s0] : -1);
                    sm.xf_pb[tid] = (short)(s1 >= 0 ? sm.rmap_prev[s1] : -1);
                }
                hs_assemble<HS_NT, 16, 1>(av, a, bl, i, kind, false, Xp, Wp, Xn, Wn);
            }
        }
        __syncthreads();
        xf.Wp = Wp;
        hs_gauss_jordan(sm, Xn, Wn, ld, n, nc, status_slot, inplace ? 1 : 0, inplace ? 2 : (hs == 0 ? 0 : 3), xf, tma_phase);
        // maps of the new result.  The elimination ran on A' = A[rl(rho)][cl(gamma)] (rl, cl = identity for an assembled A,
        // the inverse maps of the previous result for an in-place one) and left (A'^-1)[gamma][rho'] at physical
        // (perm[gamma], pinv[rho']); (A'^-1)[gamma][rho'] = (A^-1)[cl(gamma)][rl(rho')].
        if (tid == 0) {
            const unsigned km = sm.pivmin;
            kmin = min(kmin, km);
            if (kind == 0 && km != 0xffffffffu) { const double pm = __hiloint2double((int)(km << 8), 0); gsq += 1.0 / (pm * pm); }
        }
        if (tid < n) {
            const int g0 = inplace ? sm.cmap_prev[tid] : tid, r0 = inplace ? sm.rmap_prev[tid] : tid;
            sm.rmap[tid] = sm.perm[g0];
            sm.cmap[tid] = sm.pinv[r0];
        }
        __syncthreads();
    }
    if (tid < HS_NMAX) { gmaps[tid] = sm.rmap[tid]; gmaps[HS_NMAX + tid] = sm.cmap[tid]; }
    if (tid == 0 && a.pivmin) { atomicMin(a.pivmin + bl, kmin); atomicAdd(a.gsq + bl, gsq); }
    if (hs_end == a.hs_end && (a.g_out || a.P_out)) {
        const int fb = hs_out_buf(hs_end - 1);
        const cplx *Xf = fb ? X1 : X0, *Wf = fb ? W1 : W0;
        const long long os = (long long)a.nh * a.nh;
        if (a.g_out)
            for (int idx = tid; idx < n * n; idx += HS_NT) {
                const int k = idx / n, m = idx % n;
                a.g_out[bl * os + idx] = ldcg(Xf + (long long)sm.rmap[k] * ld + sm.cmap[m]);
            }
        if (a.P_out)
            for (int idx = tid; idx < n * nc; idx += HS_NT) {
                const int k = idx / nc, c = idx % nc;
                a.P_out[bl * os + (long long)k * a.nh + c] = ldcg(Wf + (long long)sm.rmap[k] * ld + c);
            }
    }
}

}  // namespace rgf
