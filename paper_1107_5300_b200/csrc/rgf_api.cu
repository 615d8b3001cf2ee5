// rgf_api.cu -- C ABI (include/rgf.h) and host orchestration of the RGF sweep on one B200.
//
// Call stack of rgf_transmission:
//   leads   : Sancho-Rubio decimation, batched over energies          (A2)  run_leads()
//   sweep   : for each slice i: assemble A_i (A1+A3) -> blocked Gauss-Jordan inverse (A4)
//             -> compact propagator GEMM (A5), batched over (device, energy)   run_sweep()
//   trace   : Gamma_R P, P^dagger (.), masked Gamma_L reduction             (A6)  run_trace()
// PyTorch is not involved: plain CUDA runtime, one stream, no CPU fallback anywhere.
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/rgf.h"
#include "gj_inverse.cuh"
#include "gj_inverse32.cuh"
#include "half_kernels.cuh"
#include "half_sweep.cuh"
#include "half_sweep_c64.cuh"
#include "lead_modes.cuh"
#include "ldos_kernels.cuh"
#include "rgf_common.cuh"
#include "sweep_kernels.cuh"
#include "zgemm.cuh"

using namespace rgf;

namespace {

struct Buf {
    void *p = nullptr;
    size_t cap = 0;
};

}  // namespace

// Workspace of the sweep.  ws[0] runs on the plan's stream: cohorts of matrices one after the other.  ws[1] has a stream
// of its own and is used by the guard pass only, whose two sweeps (from either lead) run side by side (run_dense_two_sided).
struct Ws {
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    Buf G0, G1, Nb, rowAt, orig, Pa, Pb;
    Buf H0, H1, H2, Wc, Tr, Fx0, Fx1, Fp0, Fp1, Fperm, Cp0, Cp1;                        // half-slice formulation: three compact g buffers, C P, trace scratch
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> upd_events;
    size_t upd_used = 0;
};

struct rgf_plan {
    int device = 0;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    bool has_device = false;
    int M = 0, L = 0, n_dev = 0, nh = 0;
    double t = 0.0;
    Buf onsite, bond, hop, bondc;                 // device description
    Buf E, T, status, lead_flags;                 // per call
    Buf pivmin, gsq, T_keep, redo_idx;                 // near-neutrality guard: smallest pivot per matrix, first-pass T, redone energies
    std::vector<double> guard_G, guard_Gmax;      // rms over the B half-steps / max of |t| / smallest pivot, per batch item of the last call
    double guard_tol = 1e-10;
    std::vector<Ws> ws;                           // two workspaces (see Ws)
    cudaEvent_t ev_sync[2] = {nullptr, nullptr};  // fork / join of the guard pass's second stream
    Buf jn[1];                                    // junction of the two sweeps: the block of gR the central slice couples to
    Buf gL, gR;                                   // lead surface Green's functions [n_E][M][M]
    Buf l_eps, l_eps_s, l_alpha, l_beta, l_T1, l_T2, l_T3, l_W, l_W2;   // decimation workspace
    Buf stage_in, stage_out;                      // staging for host<->device of sub-step entry points
    Buf lc_S3, lc_R;                              // run_lead_side_schur: S again and the residual of its inverse
    Buf ld_A0, ld_A1, ld_B0, ld_B1, ld_stash, ld_stashL, ld_out;   // rgf_ldos: batched G_ii work buffers, flags, the stashed gR / gL blocks, the LDOS of a chunk
    Buf lm_Q;                                     // mode-space leads: the orthogonal basis Q [nc][nc]
    Buf lead_status;                              // [n_E] bad pivot inside the lead decimation of an energy
    int lead_method = RGF_LEAD_MODE_SPACE;
    int cohort_override = 0;
    int profiling = 0;
    int formulation = RGF_FORM_HALF;
    int precision = RGF_C128;                     // of the call in progress
    bool in_sweep = false;                        // update-kernel events are taken for the sweep's inverses only
    rgf_stats stats;
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    char err[512];
    bool attrs_set = false;
};

namespace {

const char *kNoPlan = "rgf: NULL plan";

int fail(rgf_plan *p, int code, const char *fmt, ...)
{
    if (p) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(p->err, sizeof(p->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

#define CUDA_TRY(p, call)                                                                              \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess)                                                                         \
            return fail((p), e_ == cudaErrorMemoryAllocation ? RGF_ENOMEM : RGF_ECUDA, "%s failed: %s (%s:%d)", #call, \
                        cudaGetErrorString(e_), __FILE__, __LINE__);                                   \
    } while (0)

int ensure(rgf_plan *p, Buf &b, size_t bytes)
{
    if (bytes == 0) bytes = 16;
    if (b.cap >= bytes) return RGF_OK;
    if (b.p) { CUDA_TRY(p, cudaFree(b.p)); b.p = nullptr; b.cap = 0; }
    CUDA_TRY(p, cudaMalloc(&b.p, bytes));
    b.cap = bytes;
    return RGF_OK;
}

void release(Buf &b)
{
    if (b.p) cudaFree(b.p);
    b.p = nullptr;
    b.cap = 0;
}

template <typename T> T *ptr(const Buf &b) { return reinterpret_cast<T *>(b.p); }

int set_kernel_attrs(rgf_plan *p)
{
    if (p->attrs_set) return RGF_OK;
    CUDA_TRY(p, cudaFuncSetAttribute(zgemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, ZG_SMEM));
    CUDA_TRY(p, cudaFuncSetAttribute(gj_update_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, gu_smem<32>()));
    CUDA_TRY(p, cudaFuncSetAttribute(gj_update_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, gu_smem<16>()));
    CUDA_TRY(p, cudaFuncSetAttribute(gj_update_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, gu_smem<8>()));
    CUDA_TRY(p, cudaFuncSetAttribute(gj_update_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, gu_smem<4>()));
    CUDA_TRY(p, cudaFuncSetAttribute(gj_panel_kernel<16, 512, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gj_panel_smem<16, 512>(512)));
    CUDA_TRY(p, cudaFuncSetAttribute(gj_panel_kernel<8, 1024, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gj_panel_smem<8, 1024>(1024)));
    CUDA_TRY(p, cudaFuncSetAttribute(gj_panel_kernel<4, 1024, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gj_panel_smem<4, 1024>(2048)));
    CUDA_TRY(p, cudaFuncSetAttribute(gj32_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gj32_panel_smem(256)));
    CUDA_TRY(p, cudaFuncSetAttribute(gj32_update_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GU32_SMEM));
    CUDA_TRY(p, cudaFuncSetAttribute(half_sweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(HSmem)));
    CUDA_TRY(p, cudaFuncSetAttribute(half_sweep_c64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(HC64Smem)));
    CUDA_TRY(p, cudaFuncSetAttribute(gj_unpermute_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 128 * 1024));
    p->attrs_set = true;
    return RGF_OK;
}

inline int panel_width(int n) { return n <= 256 ? 32 : (n <= 512 ? 16 : (n <= 1024 ? 8 : 4)); }

int launch_zgemm(rgf_plan *p, cudaStream_t stream, const ZgemmArgs &a, int batch)
{
    if (a.Mr <= 0 || a.Nc <= 0 || batch <= 0) return RGF_OK;
    dim3 grid((a.Nc + ZG_BN - 1) / ZG_BN, (a.Mr + ZG_BM - 1) / ZG_BM, batch);
    zgemm_kernel<<<grid, ZG_THREADS, ZG_SMEM, stream>>>(a);
    p->stats.launches++;
    CUDA_TRY(p, cudaGetLastError());
    return RGF_OK;
}

// the plan's one workspace runs on the plan's stream
int ensure_ws(rgf_plan *p)
{
    if (!p->ws.empty()) return RGF_OK;
    Ws w, w2;
    w.stream = p->stream;
    CUDA_TRY(p, cudaStreamCreateWithFlags(&w2.stream, cudaStreamNonBlocking));
    w2.own_stream = true;
    for (int k = 0; k < 2; k++) CUDA_TRY(p, cudaEventCreateWithFlags(&p->ev_sync[k], cudaEventDisableTiming));
    p->ws.push_back(w);
    p->ws.push_back(w2);
    return RGF_OK;
}

// event pair bracketing one update launch (profiling level 1, sweep only)
int update_events(rgf_plan *p, Ws &w, cudaEvent_t *e0, cudaEvent_t *e1)
{
    if (w.upd_used == w.upd_events.size()) {
        if (w.upd_events.size() >= 2048) {
            CUDA_TRY(p, cudaStreamSynchronize(w.stream));
            for (size_t q = 0; q < w.upd_used; q++) {
                float ms = 0.f;
                cudaEventElapsedTime(&ms, w.upd_events[q].first, w.upd_events[q].second);
                p->stats.ms_inverse_update += ms;
            }
            w.upd_used = 0;
        } else {
            cudaEvent_t a, b;
            CUDA_TRY(p, cudaEventCreate(&a));
            CUDA_TRY(p, cudaEventCreate(&b));
            w.upd_events.push_back(std::make_pair(a, b));
        }
    }
    *e0 = w.upd_events[w.upd_used].first;
    *e1 = w.upd_events[w.upd_used].second;
    w.upd_used++;
    return RGF_OK;
}

void drain_update_events(rgf_plan *p)
{
    for (Ws &w : p->ws) {
        for (size_t q = 0; q < w.upd_used; q++) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, w.upd_events[q].first, w.upd_events[q].second) == cudaSuccess)
                p->stats.ms_inverse_update += ms;
        }
        w.upd_used = 0;
    }
}

// workspace of stream w for inverting `batch` n x n matrices
int ensure_inverse_ws(rgf_plan *p, Ws &w, int n, int batch)
{
    int B = panel_width(n), rc;
    if ((rc = ensure(p, w.Nb, sizeof(cplx) * (size_t)n * B * batch))) return rc;
    if ((rc = ensure(p, w.rowAt, sizeof(int) * (size_t)n * batch))) return rc;
    if ((rc = ensure(p, w.orig, sizeof(int) * (size_t)n * batch))) return rc;
    return RGF_OK;
}

// generic path (256 < n <= 2048): panels of 16, 8 or 4 columns, ping-pong X -> Y (rows never move); *result = buffer with the inverse
template <int B, int NT, int ROWS>
int inverse_generic(rgf_plan *p, Ws &w, cplx *G, cplx *Galt, int n, int batch, int *status, long long gb, cplx **result)
{
    cplx *Nb = ptr<cplx>(w.Nb);
    int *orig = ptr<int>(w.orig), *rowAt = ptr<int>(w.rowAt);
    cplx *X = G, *Y = Galt;
    for (int k0 = 0; k0 < n; k0 += B) {
        gj_panel_kernel<B, NT, ROWS><<<batch, NT, gj_panel_smem<B, NT>(n), w.stream>>>(X, Y, gb, n, k0, Nb, rowAt, orig, status);
        p->stats.launches++;
        dim3 grid((n + GU_BN - 1) / GU_BN, (n + GU_BM - 1) / GU_BM, batch);
        gj_update_kernel<B><<<grid, GU_THREADS, gu_smem<B>(), w.stream>>>(X, Y, gb, n, k0, Nb, rowAt);
        p->stats.launches++;
        CUDA_TRY(p, cudaGetLastError());
        std::swap(X, Y);
    }
    int nw = n > 512 ? 4 : 8;
    dim3 grid((n + nw - 1) / nw, batch);
    gj_unpermute_kernel<<<grid, nw * 32, (size_t)nw * n * sizeof(cplx), w.stream>>>(X, gb, n, orig);
    p->stats.launches++;
    CUDA_TRY(p, cudaGetLastError());
    *result = X;
    return RGF_OK;
}

// Inverse of `batch` n x n matrices stored at G (stride n*n).  Galt is a second buffer of the same
// size; *result is G or Galt, whichever holds the inverse (every path ping-pongs between the two).
// status[b] is set to 1 on a zero / non-finite pivot.
int run_inverse(rgf_plan *p, Ws &w, cplx *G, cplx *Galt, int n, int batch, int *status, cplx **result, long long stride = 0)
{
    const long long gb = stride > 0 ? stride : (long long)n * n;
    if (n > 2048) return fail(p, RGF_EUNSUPPORTED, "matrix size %d > 2048 is not supported in this version", n);
    int *orig = ptr<int>(w.orig);
    const int total = n * batch;
    gj_init_orig_kernel<<<(total + 255) / 256, 256, 0, w.stream>>>(orig, n, total);
    p->stats.launches++;
    if (n > 1024) return inverse_generic<4, 1024, 2>(p, w, G, Galt, n, batch, status, gb, result);
    if (n > 512) return inverse_generic<8, 1024, 1>(p, w, G, Galt, n, batch, status, gb, result);
    if (n > 256) return inverse_generic<16, 512, 1>(p, w, G, Galt, n, batch, status, gb, result);
    cplx *X = G, *Y = Galt, *Mult = ptr<cplx>(w.Nb);
    int *rowAt = ptr<int>(w.rowAt);
    for (int k0 = 0; k0 < n; k0 += G32_B) {
        gj32_panel_kernel<<<batch, G32_NT, gj32_panel_smem(n), w.stream>>>(X, Y, gb, n, k0, Mult, rowAt, orig, status);
        p->stats.launches++;
        if (n > G32_B) {
            dim3 grid((n + GU32_BN - 1) / GU32_BN, (n + GU32_BM - 1) / GU32_BM, batch);
            const bool timed = p->profiling > 0 && p->in_sweep;
            cudaEvent_t e0 = nullptr, e1 = nullptr;
            if (timed) {
                int rc = update_events(p, w, &e0, &e1);
                if (rc) return rc;
                CUDA_TRY(p, cudaEventRecord(e0, w.stream));
            }
            gj32_update_kernel<<<grid, GU32_THREADS, GU32_SMEM, w.stream>>>(X, Y, gb, n, k0, Mult, rowAt);
            if (timed) CUDA_TRY(p, cudaEventRecord(e1, w.stream));
            p->stats.launches++;
            if (p->in_sweep) p->stats.launches_inverse_update++;
        }
        CUDA_TRY(p, cudaGetLastError());
        std::swap(X, Y);
    }
    dim3 grid((n + 7) / 8, batch);
    gj32_unpermute_kernel<<<grid, 256, 0, w.stream>>>(X, Y, gb, n, orig);
    p->stats.launches++;
    CUDA_TRY(p, cudaGetLastError());
    *result = Y;
    return RGF_OK;
}

}  // namespace

namespace {

// A2. Lead surface Green's functions g_L (slice -1) and g_R (slice L) for n_E energies (BASELINE.json:north_star item 4).
// side -1: V_a = t diag(m_{-2}), V_b = t diag(m_{-1});  side +1: V_a = t diag(m_L), V_b = t diag(m_{L+1}).

// ------------------------------------------------------------------------------------------
// A2.  Sancho-Rubio decimation of the clean two-slice lead cell (pa, pb = slice indices of the cell, V_a = t diag(m_pa)
// inside the cell, V_b = t diag(m_pb) to the next cell) for n_E energies; writes the surface Green's function on the
// atoms that bond to the device into g_out [n_E][M][M] (zero elsewhere).
//   g = (z - eps)^-1; eps_s += (towards the bulk); eps += a g b + b g a; a <- a g a; b <- b g b   until max|a| < 1e-14 eV
// (1) alpha = h01 lives on the block (o, e), beta = alpha^T on (e, o) and the corrections of eps on X = (o, o) and
//     Y = (e, e), where e / o are the nc = M/2 atoms of the cell's first / second slice that bond to the neighbouring
//     cells (parity of pb) -- alpha g alpha etc. never leave these blocks -- so the iteration is carried on nc x nc
//     matrices and consumes only the corner blocks g[e,e], g[e,o], g[o,o] of the cell's inverse.
// (2) beta = alpha^T is kept structurally (only alpha is iterated) and g, X, Y are symmetrised: the decimation
//     squares alpha while |alpha| is O(1..100) for ~30 iterations and amplifies an antisymmetric rounding component
//     until it diverges at some energies (E = 0.4637 eV at M = 244 with alpha and beta iterated separately).
// (3) The corner blocks come either from the pivoted inverse of the whole 2M x 2M cell (dense = true) or from the
//     pivoted inverse of the 2nc x 2nc Schur complement on (e, o): the other atoms f (first slice) and b (second) bond
//     pairwise, f_j -- b_j with t, and to nothing else among themselves, so their block is [[z, -t], [-t, z]] (x) I
//     with the closed inverse [[z, t], [t, z]] / (z^2 - t^2) and
//         S = [[z - Y - k1 K, -k2 K], [-k2 K, z - X - k1 K]],  k1 = z / (z^2 - t^2),  k2 = t / (z^2 - t^2),
//     K[r][c] = t^2 * #(atoms adjacent to both corner atoms r and c): 8x fewer flops; resonant only at E = +-t, where
//     the caller takes the dense route.  The inverse of S gets one Newton step (the decimation amplifies its residual).
// ------------------------------------------------------------------------------------------
constexpr double kGuardC = 1.5e-16;        // estimated |dT| of the half-slice cut = kGuardC G_rms^2 min(1, T)
constexpr double kLeadTol = 1e-14;
constexpr int kLeadMaxIt = 64;

int run_lead_side(rgf_plan *p, int n_E, double eta, int side, int pa, int pb, bool dense, cplx *g_out, int *iters_out, int *n_open_out)
{
    const int M = p->M, qc = pb & 1, nc = half_count(M, qc), N = dense ? 2 * M : 2 * nc;
    if (N > 2048) return fail(p, RGF_EUNSUPPORTED, "lead decimation needs a %d x %d inverse; not supported in this version", N, N);
    const long long CC = (long long)nc * nc, NN = (long long)N * N;
    int rc;
    Ws &w = p->ws[0];
    Buf *cb[] = {&p->l_alpha, &p->l_beta, &p->l_T1, &p->l_T2, &p->l_T3, &p->l_eps, &p->l_eps_s, &p->stage_in};
    for (Buf *b : cb) if ((rc = ensure(p, *b, sizeof(cplx) * CC * n_E))) return rc;
    if ((rc = ensure(p, p->l_W, sizeof(cplx) * NN * n_E))) return rc;
    if ((rc = ensure(p, p->l_W2, sizeof(cplx) * NN * n_E))) return rc;
    if ((rc = ensure_inverse_ws(p, w, N, n_E))) return rc;
    cplx *a = ptr<cplx>(p->l_alpha), *b = ptr<cplx>(p->l_beta), *X = ptr<cplx>(p->l_eps), *Y = ptr<cplx>(p->l_eps_s);
    cplx *T1 = ptr<cplx>(p->l_T1), *T2 = ptr<cplx>(p->l_T2), *an = ptr<cplx>(p->l_T3);
    cplx *Sacc = ptr<cplx>(p->stage_in);          // surface accumulator: X_s (right lead, side > 0) or Y_s (left lead)
    cplx *S = ptr<cplx>(p->l_W), *S2 = ptr<cplx>(p->l_W2), *g = nullptr;
    int *flags = ptr<int>(p->lead_flags), *n_open = flags + n_E;
    int *status = ptr<int>(p->lead_status); // a bad pivot in the lead marks the energy: every device of it (fill_nan_kernel)
    const double *E = ptr<double>(p->E);
    dim3 gc((unsigned)std::min<long long>((CC + 255) / 256, 256), n_E), gs((unsigned)std::min<long long>((NN + 255) / 256, 2048), n_E);
    lead_half_init_kernel<<<gc, 256, 0, p->stream>>>(a, b, X, Y, Sacc, nc, p->t);
    p->stats.launches++;
    // position of the corner blocks inside g (N x N): element (r, c) of block (u, v) at g[(off_u + r rs) N + off_v + c rs]
    const int rs = dense ? 2 : 1, off_e = dense ? qc : 0, off_o = dense ? M + qc : nc;
    // C (nc x nc, contiguous per energy) = A B with A either a corner block of g (strided) or a compact matrix
    auto gemm = [&](const cplx *A, long long a_rs, long long a_cs, long long a_batch, const cplx *B, cplx *C) -> int {
        ZgemmArgs z;
        memset(&z, 0, sizeof(z));
        z.A = A; z.a_batch = a_batch; z.a_rs = a_rs; z.a_cs = a_cs; z.kmask_div = 1;
        z.B = B; z.b_batch = CC; z.ldb = nc;
        z.C = C; z.c_batch = CC; z.ldc = nc;
        z.Mr = z.Nc = z.K = nc;
        z.alpha = cmake(1.0, 0.0);
        return launch_zgemm(p, p->stream, z, n_E);
    };
    auto gblock = [&](const cplx *G, int off_r, int off_c) { return G + (long long)off_r * N + off_c; };
    // Schur route: one Newton step g <- sym(g + g (I - S g)).  Measured against an 80-bit reference (M = 128,
    // E = 0.2549 eV): surface Green's function off by 3.3e-10 with the plain inverse, 4.5e-11 with g symmetrised,
    // 1.1e-11 with the Newton step on top (the level of the dense route).  S is assembled a second time (the inverse
    // consumed it).
    cplx *S3 = nullptr, *Rr = nullptr;
    if (!dense) {
        if ((rc = ensure(p, p->lc_S3, sizeof(cplx) * NN * n_E))) return rc;
        if ((rc = ensure(p, p->lc_R, sizeof(cplx) * NN * n_E))) return rc;
        S3 = ptr<cplx>(p->lc_S3); Rr = ptr<cplx>(p->lc_R);
    }
    auto gemmN = [&](const cplx *A, const cplx *B, cplx *C) -> int {
        ZgemmArgs z;
        memset(&z, 0, sizeof(z));
        z.A = A; z.a_batch = NN; z.a_rs = N; z.a_cs = 1; z.kmask_div = 1;
        z.B = B; z.b_batch = NN; z.ldb = N;
        z.C = C; z.c_batch = NN; z.ldc = N;
        z.Mr = z.Nc = z.K = N;
        z.alpha = cmake(1.0, 0.0);
        return launch_zgemm(p, p->stream, z, n_E);
    };
    // g = (z - eps)^-1 restricted as needed, symmetric; Xc / Yc = corrections on (o, o) / (e, e) (NULL = none)
    auto cell_inverse = [&](const cplx *Xc, const cplx *Yc) -> int {
        int r2;
        if (dense) {
            lead_cell_assemble_kernel<<<gs, 256, 0, p->stream>>>(S, Xc, Yc, nc, M, qc, pa, p->t, E, eta);
            p->stats.launches++;
            if ((r2 = run_inverse(p, w, S, S2, N, n_E, status, &g))) return r2;
            lead_half_symmetrize_kernel<<<gs, 256, 0, p->stream>>>(g, N);
            p->stats.launches++;
            return RGF_OK;
        }
        lead_schur_assemble_kernel<<<gs, 256, 0, p->stream>>>(S, Xc, Yc, nc, M, qc, p->t, E, eta);
        p->stats.launches++;
        if ((r2 = run_inverse(p, w, S, S2, N, n_E, status, &g))) return r2;
        lead_schur_assemble_kernel<<<gs, 256, 0, p->stream>>>(S3, Xc, Yc, nc, M, qc, p->t, E, eta);
        p->stats.launches++;
        if ((r2 = gemmN(S3, g, Rr))) return r2;                       // S g
        lead_half_residual_kernel<<<gs, 256, 0, p->stream>>>(Rr, N);  // I - S g
        p->stats.launches++;
        if ((r2 = gemmN(g, Rr, S3))) return r2;                       // g (I - S g)   (S3 as scratch)
        lead_half_correct_kernel<<<gs, 256, 0, p->stream>>>(g, S3, N);
        p->stats.launches++;
        return RGF_OK;
    };
    int it = 0, open = n_E;
    for (it = 0; it < kLeadMaxIt; it++) {
        CUDA_TRY(p, cudaMemsetAsync(n_open, 0, sizeof(int), p->stream));
        lead_converged_kernel<<<n_E, 256, 0, p->stream>>>(a, a, nc, kLeadTol, flags, n_open);
        p->stats.launches++;
        CUDA_TRY(p, cudaMemcpyAsync(&open, n_open, sizeof(int), cudaMemcpyDeviceToHost, p->stream));
        CUDA_TRY(p, cudaStreamSynchronize(p->stream));
        if (open == 0) break;
        if ((rc = cell_inverse(X, Y))) return rc;
        const long long grs = (long long)rs * N;
        lead_half_transpose_kernel<<<gc, 256, 0, p->stream>>>(b, a, nc);                 // b = a^T (= beta)
        p->stats.launches++;
        if ((rc = gemm(gblock(g, off_e, off_e), grs, rs, NN, b, T1))) return rc;        // g[e,e] a^T
        if ((rc = gemm(a, nc, 1, CC, T1, T2))) return rc;                               // Tx = a g[e,e] a^T   -> (o, o)
        if ((rc = gemm(gblock(g, off_o, off_o), grs, rs, NN, a, T1))) return rc;        // g[o,o] a
        if ((rc = gemm(b, nc, 1, CC, T1, an))) return rc;                               // Ty = a^T g[o,o] a   -> (e, e)   (an as scratch)
        lead_half_accumulate_kernel<<<gc, 256, 0, p->stream>>>(X, Y, Sacc, T2, an, nc, side);
        p->stats.launches++;
        if ((rc = gemm(gblock(g, off_e, off_o), grs, rs, NN, a, T1))) return rc;        // g[e,o] a
        if ((rc = gemm(a, nc, 1, CC, T1, an))) return rc;                               // a g[e,o] a
        std::swap(a, an);
    }
    // surface block of (z - eps_s)^-1: (o, o) with Y_s for the left lead, (e, e) with X_s for the right lead
    if ((rc = cell_inverse(side > 0 ? Sacc : nullptr, side > 0 ? nullptr : Sacc))) return rc;
    CUDA_TRY(p, cudaMemsetAsync(g_out, 0, sizeof(cplx) * (size_t)M * M * n_E, p->stream));
    const int off_s = side > 0 ? off_e : off_o;
    lead_half_scatter_kernel<<<gc, 256, 0, p->stream>>>(g_out, gblock(g, off_s, off_s), M, nc, qc, rs * N, rs, NN);
    p->stats.launches++;
    CUDA_TRY(p, cudaGetLastError());
    if (iters_out) *iters_out = it;
    if (n_open_out) *n_open_out = open;
    return RGF_OK;
}

// true if the closed middle inverse of the Schur route is safely away from its resonance E = +-t
bool schur_leads_ok(rgf_plan *p, int n_E)
{
    std::vector<double> h(n_E);
    if (cudaMemcpyAsync(h.data(), p->E.p, sizeof(double) * (size_t)n_E, cudaMemcpyDeviceToHost, p->stream) != cudaSuccess) return false;
    if (cudaStreamSynchronize(p->stream) != cudaSuccess) return false;
    const double t2 = p->t * p->t;
    for (double e : h) if (std::fabs(e * e - t2) < 0.02 * t2) return false;
    return p->lead_method == RGF_LEAD_CELL_SCHUR && p->M >= 4;
}

// A2 in mode space (lead_modes.cuh): closed form per transverse mode + one real x complex product per energy
int run_lead_modes(rgf_plan *p, int n_E, double eta, int qc, cplx *g_out)
{
    const int M = p->M, nc = half_count(M, qc);
    int rc;
    if ((rc = ensure(p, p->lm_Q, sizeof(double) * (size_t)nc * nc))) return rc;
    lead_modes_basis_kernel<<<std::min((nc * nc + 255) / 256, 1024), 256, 0, p->stream>>>(ptr<double>(p->lm_Q), M, nc, qc);
    CUDA_TRY(p, cudaMemsetAsync(g_out, 0, sizeof(cplx) * (size_t)M * M * n_E, p->stream));
    for (int e0 = 0; e0 < n_E; e0 += 32768) {
        const int ne = std::min(32768, n_E - e0);
        dim3 grid((nc + 15) / 16, (nc + 15) / 16, ne);
        lead_modes_kernel<<<grid, 256, 0, p->stream>>>(g_out + (size_t)e0 * M * M, ptr<double>(p->lm_Q), M, nc, qc, p->t,
                                                      ptr<double>(p->E) + e0, eta);
        p->stats.launches++;
    }
    p->stats.launches++;
    CUDA_TRY(p, cudaGetLastError());
    return RGF_OK;
}

// both leads; for even L the two cells have the same bond parities and g_R = g_L exactly
int run_leads(rgf_plan *p, int n_E, double eta, int *n_open_out)
{
    const int M = p->M, L = p->L;
    int rc, itL = 0, itR = 0, openL = 0, openR = 0;
    const size_t MMb = sizeof(cplx) * (size_t)M * M * n_E;
    if ((rc = ensure(p, p->gL, MMb))) return rc;
    if ((rc = ensure(p, p->lead_status, sizeof(int) * (size_t)n_E))) return rc;
    if ((rc = ensure(p, p->lead_flags, sizeof(int) * (size_t)(n_E + 4)))) return rc;
    CUDA_TRY(p, cudaMemsetAsync(p->lead_status.p, 0, sizeof(int) * (size_t)n_E, p->stream));
    CUDA_TRY(p, cudaMemsetAsync(p->lead_flags.p, 0, sizeof(int) * (size_t)(n_E + 4), p->stream));
    if (p->lead_method == RGF_LEAD_MODE_SPACE) {
        if ((rc = run_lead_modes(p, n_E, eta, 1, ptr<cplx>(p->gL)))) return rc;
        if ((L & 1) != 0) {
            if ((rc = ensure(p, p->gR, MMb))) return rc;
            if ((rc = run_lead_modes(p, n_E, eta, (L - 1) & 1, ptr<cplx>(p->gR)))) return rc;
        }
        p->stats.lead_iterations = 0;
        if (n_open_out) *n_open_out = 0;
        return RGF_OK;
    }
    const bool dense = !schur_leads_ok(p, n_E);
    if ((rc = run_lead_side(p, n_E, eta, -1, -2, -1, dense, ptr<cplx>(p->gL), &itL, &openL))) return rc;
    if ((L & 1) == 0) {
        itR = itL; openR = 0;      // g_R aliases g_L (see pR() below)
    } else {
        if ((rc = ensure(p, p->gR, MMb))) return rc;
        if ((rc = run_lead_side(p, n_E, eta, +1, L, L + 1, dense, ptr<cplx>(p->gR), &itR, &openR))) return rc;
    }
    p->stats.lead_iterations = std::max(itL, itR);
    if (n_open_out) *n_open_out = openL + openR;
    return RGF_OK;
}

inline const cplx *lead_gR(const rgf_plan *p) { return (p->L & 1) == 0 ? ptr<cplx>(p->gL) : ptr<cplx>(p->gR); }

inline bool use_fused(const rgf_plan *p);
int choose_cohort(const rgf_plan *p, int batch)
{
    if (use_fused(p) && p->precision == RGF_C128) return batch;      // fused kernel: rgf_set_cohort bounds the units per launch instead
    if (p->cohort_override > 0) return std::min(p->cohort_override, batch);
    return batch;                                         // one cohort
}

int ensure_sweep_ws(rgf_plan *p, Ws &w, int cohort)
{
    int rc;
    const int M = p->M, nh = p->nh;
    if ((rc = ensure(p, w.G0, sizeof(cplx) * (size_t)M * M * cohort))) return rc;
    if ((rc = ensure(p, w.G1, sizeof(cplx) * (size_t)M * M * cohort))) return rc;
    if ((rc = ensure(p, w.Pa, sizeof(cplx) * (size_t)nh * nh * cohort))) return rc;
    if ((rc = ensure(p, w.Pb, sizeof(cplx) * (size_t)nh * nh * cohort))) return rc;
    return ensure_inverse_ws(p, w, M, cohort);
}

// A3-A5 for the cohort [bz0, bz0+nb) on workspace w: slices 0..nslices-1.  On return *G_out holds
// g_{nslices-1}, *Galt_out is the other (free) M x M buffer and *Pcur_out the compact propagator.
int run_sweep_cohort(rgf_plan *p, Ws &w, int n_E, double eta, int bz0, int nb, int nslices, cplx **G_out, cplx **Galt_out,
                     cplx **Pcur_out)
{
    const int M = p->M, L = p->L, nh = p->nh;
    int rc;
    cplx *G = ptr<cplx>(w.G0), *Galt = ptr<cplx>(w.G1), *Pcur = ptr<cplx>(w.Pa), *Pnext = ptr<cplx>(w.Pb);
    int *status = ptr<int>(p->status) + bz0;
    const double *E = ptr<double>(p->E);
    dim3 ag((unsigned)std::min<long long>(((long long)M * M + 255) / 256, 2048), nb);
    for (int i = 0; i < nslices; i++) {
        assemble_kernel<<<ag, 256, 0, w.stream>>>(G, M, L, i, n_E, bz0, E, eta, p->t, ptr<double>(p->onsite),
                                                 ptr<uint8_t>(p->bond), ptr<uint8_t>(p->hop), ptr<cplx>(p->gL), lead_gR(p));
        p->stats.launches++;
        cplx *res = nullptr;
        if ((rc = run_inverse(p, w, G, Galt, M, nb, status, &res))) return rc;
        if (res != G) std::swap(G, Galt);
        if (i == 0) {
            dim3 pg((unsigned)std::min((nh * nh + 255) / 256, 1024), nb);
            propagator_start_kernel<<<pg, 256, 0, w.stream>>>(G, Pcur, M, nh);
            p->stats.launches++;
        } else {
            // P_i[S_i, :] = t * g_i[S_i, S_{i-1}] diag(m'_{i-1}) P_{i-1}[S_{i-1}, :]   (Eq. 5)
            const int pi = i & 1, pp = (i - 1) & 1;
            ZgemmArgs a;
            memset(&a, 0, sizeof(a));
            a.A = G + (long long)pi * M + pp; a.a_batch = (long long)M * M; a.a_rs = 2LL * M; a.a_cs = 2;
            a.kmask = ptr<uint8_t>(p->bondc) + (long long)i * nh;                              // m'_{i-1} compact
            a.kmask_batch = (long long)(L + 1) * nh; a.kmask_div = n_E; a.kmask_b0 = bz0;
            a.B = Pcur; a.b_batch = (long long)nh * nh; a.ldb = nh;
            a.C = Pnext; a.c_batch = (long long)nh * nh; a.ldc = nh;
            a.Mr = (M - pi + 1) / 2; a.K = (M - pp + 1) / 2; a.Nc = M / 2;
            a.alpha = cmake(p->t, 0.0);
            if ((rc = launch_zgemm(p, w.stream, a, nb))) return rc;
            std::swap(Pcur, Pnext);
        }
    }
    CUDA_TRY(p, cudaGetLastError());
    *G_out = G; *Galt_out = Galt; *Pcur_out = Pcur;
    return RGF_OK;
}

int run_trace_cohort(rgf_plan *p, Ws &w, int n_E, int bz0, int nb, cplx *scratch, cplx *Pcur);

// The dense formulation swept from BOTH leads at once, for the guard pass: a handful of matrices, where the time is the
// sequential latency of the slices (0.5 ms each), not throughput.  Left chain (plan's stream): slices 0 .. m with
// P_m = G^L_{m,0}; right chain (second stream, side by side on the idle SMs): slices L-1 .. c+1, c = m + 1, with
// Q = G^R_{c+1,L-1}; both are lead-connected, hence as stable as the one-sided sweep.  They meet at the central slice c, which
// is added like any slice of the one-sided sweep, the right part standing in for a lead:
//     G_cc = (z - H_c - V_m gL_m V_m - V_c gR_{c+1} V_c)^-1,   G_{c,0} = G_cc V_m P_m,   G_{L-1,0} = Q^T V_c G_{c,0}   (G = G^T)
// (Dyson's equation, Eq. 3), then the trace as usual.  Every block that is multiplied connects the two
// sublattices; the closed form that joins the two surfaces directly, (1 - gL V gR V)^-1, contains the same-sublattice blocks
// of two terminated halves, which diverge like 1/E towards charge neutrality, and lost 5e-9 at |E| = 4e-3 eV (measured).
// Half the sequential steps.  Covers the cohort [bz0, bz0 + nb); writes p->T.
int run_dense_two_sided(rgf_plan *p, int n_E, double eta, int bz0, int nb)
{
    const int M = p->M, L = p->L, nh = p->nh, m = L / 2 - 1;
    Ws &wl = p->ws[0], &wr = p->ws[1];
    int rc;
    if ((rc = ensure_sweep_ws(p, wl, nb)) || (rc = ensure_sweep_ws(p, wr, nb))) return rc;
    const size_t hb = sizeof(cplx) * (size_t)nh * nh * nb;
    for (Buf &b : p->jn) if ((rc = ensure(p, b, hb))) return rc;
    int *status = ptr<int>(p->status) + bz0;
    const double *E = ptr<double>(p->E);
    const long long hs = (long long)nh * nh, MM = (long long)M * M;
    cplx *GL = ptr<cplx>(wl.G0), *GLalt = ptr<cplx>(wl.G1), *Pcur = ptr<cplx>(wl.Pa), *Pnext = ptr<cplx>(wl.Pb);
    cplx *GR = ptr<cplx>(wr.G0), *GRalt = ptr<cplx>(wr.G1), *Qcur = ptr<cplx>(wr.Pa), *Qnext = ptr<cplx>(wr.Pb);
    dim3 ag((unsigned)std::min<long long>((MM + 255) / 256, 2048), nb), pg((unsigned)std::min((nh * nh + 255) / 256, 1024), nb);
    const int nR = half_count(M, (L - 1) & 1);
    auto masked_gemm = [&](cudaStream_t st, const cplx *A, long long a_batch, long long a_rs, long long a_cs, int mask_row, const cplx *B,
                           cplx *C, int Mr, int K, int Nc, double alpha) -> int {
        ZgemmArgs a;
        memset(&a, 0, sizeof(a));
        a.A = A; a.a_batch = a_batch; a.a_rs = a_rs; a.a_cs = a_cs; a.kmask_div = 1;
        if (mask_row >= 0) {
            a.kmask = ptr<uint8_t>(p->bondc) + (long long)mask_row * nh;
            a.kmask_batch = (long long)(L + 1) * nh; a.kmask_div = n_E; a.kmask_b0 = bz0;
        }
        a.B = B; a.b_batch = hs; a.ldb = nh;
        a.C = C; a.c_batch = hs; a.ldc = nh;
        a.Mr = Mr; a.K = K; a.Nc = Nc; a.alpha = cmake(alpha, 0.0);
        return launch_zgemm(p, st, a, nb);
    };
    auto left_step = [&](int i) -> int {
        assemble_kernel<<<ag, 256, 0, wl.stream>>>(GL, M, L, i, n_E, bz0, E, eta, p->t, ptr<double>(p->onsite), ptr<uint8_t>(p->bond),
                                                  ptr<uint8_t>(p->hop), ptr<cplx>(p->gL), lead_gR(p));
        p->stats.launches++;
        cplx *res = nullptr;
        int r2 = run_inverse(p, wl, GL, GLalt, M, nb, status, &res);
        if (r2) return r2;
        if (res != GL) std::swap(GL, GLalt);
        if (i == 0) {
            propagator_start_kernel<<<pg, 256, 0, wl.stream>>>(GL, Pcur, M, nh);
            p->stats.launches++;
            return RGF_OK;
        }
        const int pi = i & 1, pp = (i - 1) & 1;      // P_i[S_i, :] = t g_i[S_i, S_{i-1}] m'_{i-1} P_{i-1}
        r2 = masked_gemm(wl.stream, GL + (long long)pi * M + pp, MM, 2LL * M, 2, i, Pcur, Pnext, half_count(M, pi), half_count(M, pp), M / 2, p->t);
        std::swap(Pcur, Pnext);
        return r2;
    };
    auto right_step = [&](int i) -> int {
        assemble_right_kernel<<<ag, 256, 0, wr.stream>>>(GR, M, L, i, n_E, bz0, E, eta, p->t, ptr<double>(p->onsite), ptr<uint8_t>(p->bond),
                                                        ptr<uint8_t>(p->hop), lead_gR(p));
        p->stats.launches++;
        cplx *res = nullptr;
        int r2 = run_inverse(p, wr, GR, GRalt, M, nb, status, &res);
        if (r2) return r2;
        if (res != GR) std::swap(GR, GRalt);
        const int pr = (i - 1) & 1, pc = i & 1;      // rows: atoms bonded to slice i - 1; Q_i = t gR_i[., S_i] m'_i Q_{i+1}
        if (i == L - 1) {
            block_extract_kernel<<<pg, 256, 0, wr.stream>>>(GR, Qcur, M, nh, pr, pc);
            p->stats.launches++;
            return RGF_OK;
        }
        r2 = masked_gemm(wr.stream, GR + (long long)pr * M + pc, MM, 2LL * M, 2, i + 1, Qcur, Qnext, half_count(M, pr), half_count(M, pc), nR, p->t);
        std::swap(Qcur, Qnext);
        return r2;
    };
    CUDA_TRY(p, cudaEventRecord(p->ev_sync[0], p->stream));
    CUDA_TRY(p, cudaStreamWaitEvent(wr.stream, p->ev_sync[0], 0));
    const int nl = m + 1, nr = L - 2 - m;          // the central slice c = m + 1 belongs to neither chain
    for (int s = 0; s < std::max(nl, nr); s++) {
        if (s < nl && (rc = left_step(s))) return rc;
        if (s < nr && (rc = right_step(L - 1 - s))) return rc;
    }
    CUDA_TRY(p, cudaGetLastError());
    CUDA_TRY(p, cudaEventRecord(p->ev_sync[1], wr.stream));
    CUDA_TRY(p, cudaStreamWaitEvent(p->stream, p->ev_sync[1], 0));
    // ---- central slice c and the junction, on the plan's stream
    const int c = m + 1, pc = c & 1, pm = m & 1;
    cplx *J0 = ptr<cplx>(p->jn[0]);
    block_extract_kernel<<<pg, 256, 0, wl.stream>>>(GR, J0, M, nh, pc, pc);                // the block of gR_{c+1} that V_c keeps
    ldos_assemble_kernel<<<ag, 256, 0, wl.stream>>>(GLalt, M, L, nh, c, n_E, bz0, E, eta, p->t, ptr<double>(p->onsite), ptr<uint8_t>(p->bond),
                                                   ptr<uint8_t>(p->hop), 1, GL, ptr<cplx>(p->gL), 1, J0, lead_gR(p));
    p->stats.launches += 2;
    cplx *Gcc = nullptr;
    if ((rc = run_inverse(p, wl, GLalt, GL, M, nb, status, &Gcc))) return rc;
    cplx *Gfree = (Gcc == GLalt) ? GL : GLalt;
    if ((rc = masked_gemm(wl.stream, Gcc + (long long)pc * M + pm, MM, 2LL * M, 2, c, Pcur, Pnext, half_count(M, pc), half_count(M, pm), M / 2, p->t))) return rc;   // G_{c,0}
    if ((rc = masked_gemm(wl.stream, Qcur, hs, 1, nh, c + 1, Pnext, Pcur, nR, half_count(M, pc), M / 2, p->t))) return rc;        // G_{L-1,0} = t Q^T m'_c G_{c,0}
    CUDA_TRY(p, cudaGetLastError());
    return run_trace_cohort(p, wl, n_E, bz0, nb, Gfree, Pcur);
}

// ---- half-slice formulation (half_kernels.cuh): 2 half-steps per slice, each an (M/2) inverse and an (M/2)^3 GEMM ----
int ensure_sweep_ws_half(rgf_plan *p, Ws &w, int cohort)
{
    int rc;
    const int nh = p->nh;
    const size_t hb = sizeof(cplx) * (size_t)nh * nh * cohort;
    Buf *bufs[] = {&w.H0, &w.H1, &w.H2, &w.Wc, &w.Pa, &w.Pb};
    for (Buf *b : bufs) if ((rc = ensure(p, *b, hb))) return rc;
    if ((rc = ensure(p, w.Tr, 2 * hb))) return rc;
    return ensure_inverse_ws(p, w, nh, cohort);
}

// slices 0..nslices-1 of the cohort [bz0, bz0+nb); *g_out = gF of the last slice (dense n x n at stride nh*nh),
// *Pcur_out its compact propagator (rows F_i, columns B_0, ld nh)
inline bool use_fused(const rgf_plan *p) { return p->formulation == RGF_FORM_HALF && p->nh <= HS_NMAX; }

// fused path (half_sweep.cuh): one CTA per matrix runs every half-step of slices 0..nslices-1 in ONE launch
// launches half_sweep_kernel for the nb matrices described by `a` (state buffers of workspace w are set here)
int fused_launch(rgf_plan *p, Ws &w, HSweepArgs &a, int nb)
{
    int rc;
    const size_t xb = sizeof(cplx) * (size_t)a.ldn * a.ldn * nb;
    Buf *bufs[] = {&w.Fx0, &w.Fx1, &w.Fp0, &w.Fp1};
    for (Buf *b : bufs) if ((rc = ensure(p, *b, xb))) return rc;
    if ((rc = ensure(p, w.Fperm, sizeof(int) * 2 * (size_t)HS_NMAX * nb))) return rc;      // row and column maps
    a.nb = nb;
    a.X0 = ptr<cplx>(w.Fx0); a.X1 = ptr<cplx>(w.Fx1); a.P0 = ptr<cplx>(w.Fp0); a.P1 = ptr<cplx>(w.Fp1);
    a.perm = ptr<int>(w.Fperm);
    // Rounds of units: with more matrices than resident CTA slots (2 per SM) a single launch would run 512 matrices
    // as 296 + 216, the second wave half empty.  Instead every launch runs `slots` units of unit_len half-steps; unit
    // u = (matrix u % nb, chunk u / nb), so chunk c+1 of a matrix is always in a later launch than its chunk c
    // (nb > slots) and stream order is the only dependency.
    int sms = 0, occ = 0;
    CUDA_TRY(p, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p->device));
    CUDA_TRY(p, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, half_sweep_kernel, HS_NT, sizeof(HSmem)));
    int slots = std::max(1, occ) * sms;
    if (p->cohort_override > 0) slots = std::min(slots, p->cohort_override);      // rgf_set_cohort: fewer units per launch
    const bool timed = p->profiling > 0 && p->in_sweep;
    auto launch = [&](unsigned grid) -> int {
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        if (timed) {
            int rc2 = update_events(p, w, &e0, &e1);
            if (rc2) return rc2;
            CUDA_TRY(p, cudaEventRecord(e0, w.stream));
        }
        half_sweep_kernel<<<grid, HS_NT, sizeof(HSmem), w.stream>>>(a);
        if (timed) CUDA_TRY(p, cudaEventRecord(e1, w.stream));
        p->stats.launches++;
        if (p->in_sweep) p->stats.launches_inverse_update++;
        return RGF_OK;
    };
    if (nb <= slots) {
        a.unit0 = 0; a.unit_len = a.hs_end;
        if ((rc = launch((unsigned)nb))) return rc;
    } else {
        a.unit_len = std::min(a.hs_end, 64);
        const long long nchunks = (a.hs_end + a.unit_len - 1) / a.unit_len, units = nchunks * nb;
        for (long long u0 = 0; u0 < units; u0 += slots) {
            a.unit0 = (int)u0;
            if ((rc = launch((unsigned)std::min<long long>(slots, units - u0)))) return rc;
        }
    }
    CUDA_TRY(p, cudaGetLastError());
    return RGF_OK;
}

int run_sweep_cohort_fused(rgf_plan *p, Ws &w, int n_E, double eta, int bz0, int nb, int nslices, cplx **g_out, cplx **Pcur_out)
{
    const int nh = p->nh, ldn = (nh + 1) & ~1;
    int rc;
    HSweepArgs a;
    memset(&a, 0, sizeof(a));
    a.M = p->M; a.L = p->L; a.nh = nh; a.ldn = ldn; a.n_E = n_E; a.bz0 = bz0; a.eta = eta; a.t = p->t;
    a.energies = ptr<double>(p->E); a.onsite = ptr<double>(p->onsite);
    a.bond = ptr<uint8_t>(p->bond); a.hop = ptr<uint8_t>(p->hop);
    a.gL = ptr<cplx>(p->gL); a.gR = lead_gR(p);
    a.status = ptr<int>(p->status) + bz0;
    a.pivmin = p->pivmin.p ? ptr<unsigned>(p->pivmin) + bz0 : nullptr;
    a.gsq = p->gsq.p ? ptr<double>(p->gsq) + bz0 : nullptr;
    a.hs_begin = 0; a.hs_end = 2 * nslices;
    a.g_out = ptr<cplx>(w.H0); a.P_out = ptr<cplx>(w.Pa);
    if ((rc = fused_launch(p, w, a, nb))) return rc;
    *g_out = ptr<cplx>(w.H0); *Pcur_out = ptr<cplx>(w.Pa);
    return RGF_OK;
}

// complex64 sweep (half_sweep_c64.cuh): one CTA per matrix for the whole sweep, FP32 FFMA
int run_sweep_cohort_c64(rgf_plan *p, Ws &w, int n_E, double eta, int bz0, int nb, int nslices, cplx **g_out, cplx **Pcur_out)
{
    int rc;
    const size_t pb = sizeof(float2) * (size_t)HC_NMAX * HC_NMAX * nb;
    if ((rc = ensure(p, w.Cp0, pb))) return rc;
    if ((rc = ensure(p, w.Cp1, pb))) return rc;
    HC64Args a;
    memset(&a, 0, sizeof(a));
    a.M = p->M; a.L = p->L; a.nh = p->nh; a.n_E = n_E; a.bz0 = bz0; a.nb = nb; a.eta = eta; a.t = p->t;
    a.energies = ptr<double>(p->E); a.onsite = ptr<double>(p->onsite);
    a.bond = ptr<uint8_t>(p->bond); a.hop = ptr<uint8_t>(p->hop);
    a.gL = ptr<cplx>(p->gL); a.gR = lead_gR(p);
    a.P0 = ptr<float2>(w.Cp0); a.P1 = ptr<float2>(w.Cp1);
    a.status = ptr<int>(p->status) + bz0;
    a.hs_end = 2 * nslices;
    a.g_out = ptr<cplx>(w.H0); a.P_out = ptr<cplx>(w.Pa);
    half_sweep_c64_kernel<<<nb, HC_NT, sizeof(HC64Smem), w.stream>>>(a);
    p->stats.launches++;
    CUDA_TRY(p, cudaGetLastError());
    *g_out = ptr<cplx>(w.H0); *Pcur_out = ptr<cplx>(w.Pa);
    return RGF_OK;
}

int run_sweep_cohort_half(rgf_plan *p, Ws &w, int n_E, double eta, int bz0, int nb, int nslices, cplx **g_out, cplx **Pcur_out)
{
    if (p->precision == RGF_C64) return run_sweep_cohort_c64(p, w, n_E, eta, bz0, nb, nslices, g_out, Pcur_out);
    if (use_fused(p)) return run_sweep_cohort_fused(p, w, n_E, eta, bz0, nb, nslices, g_out, Pcur_out);
    const int M = p->M, L = p->L, nh = p->nh, nc = M / 2;
    const long long hs = (long long)nh * nh;
    int rc;
    cplx *gprev = ptr<cplx>(w.H0), *fa = ptr<cplx>(w.H1), *fb = ptr<cplx>(w.H2);
    cplx *Pcur = ptr<cplx>(w.Pa), *Pnext = ptr<cplx>(w.Pb), *W = ptr<cplx>(w.Wc);
    int *status = ptr<int>(p->status) + bz0;
    HalfArgs ha;
    memset(&ha, 0, sizeof(ha));
    ha.M = M; ha.L = L; ha.nh = nh; ha.n_E = n_E; ha.bz0 = bz0; ha.eta = eta; ha.t = p->t;
    ha.energies = ptr<double>(p->E); ha.onsite = ptr<double>(p->onsite);
    ha.bond = ptr<uint8_t>(p->bond); ha.hop = ptr<uint8_t>(p->hop);
    ha.gL = ptr<cplx>(p->gL); ha.gR = lead_gR(p);
    dim3 eg((unsigned)std::min((int)((hs + 255) / 256), 1024), nb);
    for (int i = 0; i < nslices; i++) {
        for (int kind = 0; kind < 2; kind++) {
            const int par = kind == 0 ? ((i + 1) & 1) : (i & 1);
            const int n = half_count(M, par);
            ha.i = i; ha.kind = kind;
            if (n == 0) continue;           // M = 1 is rejected earlier; n >= 1 always for M >= 2
            half_assemble_kernel<<<eg, 256, 0, w.stream>>>(fa, gprev, ha);
            p->stats.launches++;
            cplx *res = nullptr;
            if ((rc = run_inverse(p, w, fa, fb, n, nb, status, &res, hs))) return rc;
            // rotate: res becomes gprev, the other two are free
            cplx *other = (res == fa) ? fb : fa;
            cplx *old = gprev;
            gprev = res; fa = old; fb = other;
            if (i == 0 && kind == 0) {
                half_start_kernel<<<eg, 256, 0, w.stream>>>(Pcur, gprev, n, nh);
                p->stats.launches++;
            } else {
                half_couple_kernel<<<eg, 256, 0, w.stream>>>(W, Pcur, ha);
                p->stats.launches++;
                ZgemmArgs a;
                memset(&a, 0, sizeof(a));
                a.A = gprev; a.a_batch = hs; a.a_rs = n; a.a_cs = 1; a.kmask_div = 1;
                a.B = W; a.b_batch = hs; a.ldb = nh;
                a.C = Pnext; a.c_batch = hs; a.ldc = nh;
                a.Mr = n; a.K = n; a.Nc = nc;
                a.alpha = cmake(1.0, 0.0);
                if ((rc = launch_zgemm(p, w.stream, a, nb))) return rc;
                std::swap(Pcur, Pnext);
            }
        }
    }
    CUDA_TRY(p, cudaGetLastError());
    *g_out = gprev; *Pcur_out = Pcur;
    return RGF_OK;
}

// A6 for the cohort: T = Re Tr[Gamma_L P^dagger Gamma_R P]  (Eq. 2)
int run_trace_cohort(rgf_plan *p, Ws &w, int n_E, int bz0, int nb, cplx *scratch, cplx *Pcur)
{
    const int M = p->M, L = p->L, nh = p->nh;
    int rc;
    cplx *Gam = scratch, *Y = scratch + (size_t)nh * nh * nb;      // an M x M buffer per matrix holds both
    cplx *X = (Pcur == ptr<cplx>(w.Pa)) ? ptr<cplx>(w.Pb) : ptr<cplx>(w.Pa);
    const int pR = (L - 1) & 1, nr = (M - pR + 1) / 2, nc = M / 2;
    dim3 gg((unsigned)std::min((nh * nh + 255) / 256, 1024), nb);
    gamma_right_kernel<<<gg, 256, 0, w.stream>>>(Gam, lead_gR(p), ptr<uint8_t>(p->bond), M, L, nh, n_E, bz0, p->t);
    p->stats.launches++;
    ZgemmArgs a;
    memset(&a, 0, sizeof(a));                            // X = Gamma_R P
    a.A = Gam; a.a_batch = (long long)nh * nh; a.a_rs = nh; a.a_cs = 1; a.kmask_div = 1;
    a.B = Pcur; a.b_batch = (long long)nh * nh; a.ldb = nh;
    a.C = X; a.c_batch = (long long)nh * nh; a.ldc = nh;
    a.Mr = nr; a.K = nr; a.Nc = nc; a.alpha = cmake(1.0, 0.0);
    if ((rc = launch_zgemm(p, w.stream, a, nb))) return rc;
    memset(&a, 0, sizeof(a));                            // Y = P^dagger X
    a.A = Pcur; a.a_batch = (long long)nh * nh; a.a_rs = 1; a.a_cs = nh; a.conjA = 1; a.kmask_div = 1;
    a.B = X; a.b_batch = (long long)nh * nh; a.ldb = nh;
    a.C = Y; a.c_batch = (long long)nh * nh; a.ldc = nh;
    a.Mr = nc; a.K = nr; a.Nc = nc; a.alpha = cmake(1.0, 0.0);
    if ((rc = launch_zgemm(p, w.stream, a, nb))) return rc;
    trace_kernel<<<nb, 256, 0, w.stream>>>(Y, ptr<cplx>(p->gL), ptr<uint8_t>(p->bond), M, L, nh, n_E, bz0, p->t, ptr<double>(p->T));
    p->stats.launches++;
    CUDA_TRY(p, cudaGetLastError());
    return RGF_OK;
}

int upload_energies(rgf_plan *p, const double *energies, int n_E, double eta)
{
    if (!energies || n_E < 1) return fail(p, RGF_EINVAL, "energies NULL or n_E < 1");
    if (!(eta > 0.0) || !std::isfinite(eta)) return fail(p, RGF_EINVAL, "eta must be finite and > 0");
    int rc;
    if ((rc = ensure(p, p->E, sizeof(double) * (size_t)n_E))) return rc;
    CUDA_TRY(p, cudaMemcpyAsync(p->E.p, energies, sizeof(double) * (size_t)n_E, cudaMemcpyDefault, p->stream));
    return RGF_OK;
}

int begin_call(rgf_plan *p)
{
    if (!p) return RGF_EINVAL;
    p->err[0] = 0;
    CUDA_TRY(p, cudaSetDevice(p->device));
    int rc = ensure_ws(p);
    if (rc) return rc;
    return set_kernel_attrs(p);
}

}  // namespace

// ==========================================================================================
// Exported C ABI
// ==========================================================================================
extern "C" {

int rgf_plan_create(rgf_plan **out, int cuda_device, void *cuda_stream)
{
    if (!out) return RGF_EINVAL;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) return RGF_ECUDA;
    rgf_plan *p = new (std::nothrow) rgf_plan();
    if (!p) return RGF_ENOMEM;
    p->err[0] = 0;
    memset(&p->stats, 0, sizeof(p->stats));
    p->device = cuda_device;
    if (cudaSetDevice(cuda_device) != cudaSuccess) { delete p; return RGF_ECUDA; }
    if (cuda_stream) {
        p->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    } else {
        if (cudaStreamCreateWithFlags(&p->stream, cudaStreamNonBlocking) != cudaSuccess) { delete p; return RGF_ECUDA; }
        p->own_stream = true;
    }
    for (int i = 0; i < 5; i++)
        if (cudaEventCreate(&p->ev[i]) != cudaSuccess) { delete p; return RGF_ECUDA; }
    *out = p;
    return RGF_OK;
}

int rgf_set_device_batch(rgf_plan *p, int n_dev, int M, int L, const double *onsite, double t, const uint8_t *vacancy)
{
    int rc = begin_call(p);
    if (rc) return rc;
    if (n_dev < 1 || M < 2 || L < 1 || !onsite || !std::isfinite(t))
        return fail(p, RGF_EINVAL, "rgf_set_device: need n_dev >= 1, M >= 2, L >= 1, onsite != NULL, finite t");
    if (M > 1024) return fail(p, RGF_EUNSUPPORTED, "M = %d > 1024 is not supported in this version", M);
    const size_t nsite = (size_t)n_dev * L * M;
    // the masks are derived on the host (O(L M) bytes, once per device): bring the inputs here first
    std::vector<double> h_on(nsite);
    std::vector<uint8_t> h_vac(nsite, 0);
    CUDA_TRY(p, cudaMemcpy(h_on.data(), onsite, sizeof(double) * nsite, cudaMemcpyDefault));
    if (vacancy) CUDA_TRY(p, cudaMemcpy(h_vac.data(), vacancy, nsite, cudaMemcpyDefault));
    for (size_t k = 0; k < nsite; k++)
        if (!std::isfinite(h_on[k])) return fail(p, RGF_EINVAL, "onsite[%zu] is not finite", k);
    const int nh = (M + 1) / 2;
    std::vector<uint8_t> h_bond((size_t)n_dev * (L + 1) * M), h_hop(nsite), h_bondc((size_t)n_dev * (L + 1) * nh, 0);
    for (int d = 0; d < n_dev; d++) {
        const uint8_t *vac = h_vac.data() + (size_t)d * L * M;
        auto isvac = [&](int i, int j) { return (i >= 0 && i < L) ? vac[(size_t)i * M + j] != 0 : false; };
        for (int i = -1; i < L; i++) {
            uint8_t *bm = h_bond.data() + ((size_t)d * (L + 1) + (i + 1)) * M;
            uint8_t *bc = h_bondc.data() + ((size_t)d * (L + 1) + (i + 1)) * nh;
            for (int j = 0; j < M; j++) {
                bm[j] = (mask_bit(i, j) && !isvac(i, j) && !isvac(i + 1, j)) ? 1 : 0;
                if (mask_bit(i, j)) bc[j >> 1] = bm[j];       // j = 2k + (i & 1)
            }
        }
        for (int i = 0; i < L; i++)
            for (int j = 0; j < M; j++)
                h_hop[((size_t)d * L + i) * M + j] = (j + 1 < M && !isvac(i, j) && !isvac(i, j + 1)) ? 1 : 0;
    }
    if ((rc = ensure(p, p->onsite, sizeof(double) * nsite))) return rc;
    if ((rc = ensure(p, p->bond, h_bond.size()))) return rc;
    if ((rc = ensure(p, p->hop, h_hop.size()))) return rc;
    if ((rc = ensure(p, p->bondc, h_bondc.size()))) return rc;
    CUDA_TRY(p, cudaMemcpy(p->onsite.p, h_on.data(), sizeof(double) * nsite, cudaMemcpyHostToDevice));
    CUDA_TRY(p, cudaMemcpy(p->bond.p, h_bond.data(), h_bond.size(), cudaMemcpyHostToDevice));
    CUDA_TRY(p, cudaMemcpy(p->hop.p, h_hop.data(), h_hop.size(), cudaMemcpyHostToDevice));
    CUDA_TRY(p, cudaMemcpy(p->bondc.p, h_bondc.data(), h_bondc.size(), cudaMemcpyHostToDevice));
    p->M = M; p->L = L; p->n_dev = n_dev; p->nh = nh; p->t = t;
    p->has_device = true;
    return RGF_OK;
}

int rgf_set_device(rgf_plan *p, int M, int L, const double *onsite, double t, const uint8_t *vacancy)
{
    return rgf_set_device_batch(p, 1, M, L, onsite, t, vacancy);
}

// One pass of the hot path over the n_E energies in p->E: leads (A2), sweep (A3-A5) and trace (A6) in `formulation`.
// Writes p->T [n_dev][n_E] (NaN where an energy failed), p->status, p->lead_flags / p->lead_status, and for the fused
// kernel p->pivmin.  *lead_open = number of energies whose lead decimation did not converge.
static int transmission_pass(rgf_plan *p, int n_E, double eta, int formulation, int *lead_open_out, bool first_pass = true)
{
    int rc;
    const int batch = p->n_dev * n_E;
    if ((rc = ensure(p, p->status, sizeof(int) * (size_t)batch))) return rc;
    if ((rc = ensure(p, p->T, sizeof(double) * (size_t)batch))) return rc;
    if ((rc = ensure(p, p->pivmin, sizeof(unsigned) * (size_t)batch))) return rc;
    if ((rc = ensure(p, p->gsq, sizeof(double) * (size_t)batch))) return rc;
    CUDA_TRY(p, cudaMemsetAsync(p->gsq.p, 0, sizeof(double) * (size_t)batch, p->stream));
    CUDA_TRY(p, cudaMemsetAsync(p->status.p, 0, sizeof(int) * (size_t)batch, p->stream));
    CUDA_TRY(p, cudaMemsetAsync(p->pivmin.p, 0xff, sizeof(unsigned) * (size_t)batch, p->stream));
    const int saved_form = p->formulation;
    p->formulation = formulation;
    int lead_open = 0;
    CUDA_TRY(p, cudaEventRecord(p->ev[1], p->stream));
    nvtxRangePushA("rgf_leads");
    const long long l0 = p->stats.launches;
    rc = run_leads(p, n_E, eta, &lead_open);
    nvtxRangePop();
    if (rc) { p->formulation = saved_form; return rc; }
    p->stats.launches_leads += p->stats.launches - l0;
    CUDA_TRY(p, cudaEventRecord(p->ev[2], p->stream));
    // ---- sweep + trace, cohort after cohort
    const int cohort = choose_cohort(p, batch);
    if (first_pass) p->stats.cohort = cohort;
    const bool half = formulation != RGF_FORM_DENSE;
    Ws &w = p->ws[0];
    if ((rc = half ? ensure_sweep_ws_half(p, w, cohort) : ensure_sweep_ws(p, w, cohort))) { p->formulation = saved_form; return rc; }
    nvtxRangePushA("rgf_sweep");
    p->in_sweep = first_pass;          // the dominant kernel's events and launch count describe the first pass only
    for (int bz0 = 0; bz0 < batch && rc == RGF_OK; bz0 += cohort) {
        const int nb = std::min(cohort, batch - bz0);
        cplx *G = nullptr, *Galt = nullptr, *Pcur = nullptr;
        if (half) {
            rc = run_sweep_cohort_half(p, w, n_E, eta, bz0, nb, p->L, &G, &Pcur);
            Galt = ptr<cplx>(w.Tr);
        } else if (!first_pass && p->L >= 4) {
            rc = run_dense_two_sided(p, n_E, eta, bz0, nb);          // includes the trace
            continue;
        } else {
            rc = run_sweep_cohort(p, w, n_E, eta, bz0, nb, p->L, &G, &Galt, &Pcur);
        }
        if (rc == RGF_OK) rc = run_trace_cohort(p, w, n_E, bz0, nb, Galt, Pcur);
    }
    p->in_sweep = false;
    nvtxRangePop();
    p->formulation = saved_form;
    if (rc) return rc;
    // failed items -> NaN; a lead failure (per energy) hits every device of that energy
    fill_nan_kernel<<<(batch + 255) / 256, 256, 0, p->stream>>>(ptr<double>(p->T), ptr<int>(p->status), ptr<int>(p->lead_flags),
                                                             ptr<int>(p->lead_status), batch, n_E);
    p->stats.launches++;
    CUDA_TRY(p, cudaEventRecord(p->ev[3], p->stream));
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, p->ev[1], p->ev[2]); p->stats.ms_leads += ms;
    cudaEventElapsedTime(&ms, p->ev[2], p->ev[3]); p->stats.ms_sweep += ms;
    if (!first_pass) { float m2 = 0.f; cudaEventElapsedTime(&m2, p->ev[1], p->ev[3]); p->stats.ms_guard += m2; }
    if (lead_open_out) *lead_open_out = lead_open;
    return RGF_OK;
}

// result code of a pass from the flags it left on the device (host copies)
static int pass_result(rgf_plan *p, int n_E, int lead_open, int result)
{
    const int batch = p->n_dev * n_E;
    std::vector<int> h_status(batch), h_ls(n_E);
    CUDA_TRY(p, cudaMemcpyAsync(h_status.data(), p->status.p, sizeof(int) * (size_t)batch, cudaMemcpyDeviceToHost, p->stream));
    CUDA_TRY(p, cudaMemcpyAsync(h_ls.data(), p->lead_status.p, sizeof(int) * (size_t)n_E, cudaMemcpyDeviceToHost, p->stream));
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    if (lead_open)
        result = fail(p, RGF_ENOCONV, "lead decimation did not converge in %d iterations for %d energies", kLeadMaxIt, lead_open);
    for (int e = 0; e < n_E; e++)
        if (h_ls[e]) { result = fail(p, RGF_ESINGULAR, "zero or non-finite pivot in the lead decimation of energy %d", e); break; }
    for (int b = 0; b < batch; b++)
        if (h_status[b]) { result = fail(p, RGF_ESINGULAR, "zero or non-finite pivot (first at batch item %d)", b); break; }
    return result;
}

int rgf_transmission(rgf_plan *p, const double *energies, int n_E, double eta, int precision, double *T_out)
{
    int rc = begin_call(p);
    if (rc) return rc;
    if (!p->has_device) return fail(p, RGF_ESTATE, "rgf_transmission before rgf_set_device");
    if (!T_out) return fail(p, RGF_EINVAL, "T_out is NULL");
    if (precision != RGF_C128 && precision != RGF_C64) return fail(p, RGF_EINVAL, "precision must be RGF_C128 or RGF_C64");
    if (precision == RGF_C64 && (p->formulation != RGF_FORM_HALF || p->nh > HC_NMAX))
        return fail(p, RGF_EUNSUPPORTED, "the complex64 sweep is built for RGF_FORM_HALF and M <= 256 only");
    if (n_E >= 1 && (long long)p->n_dev * n_E > 65535)
        return fail(p, RGF_EUNSUPPORTED, "n_dev * n_E = %lld > 65535 batch items per call: split the energy grid", (long long)p->n_dev * n_E);
    p->precision = precision;
    memset(&p->stats, 0, sizeof(p->stats));
    p->ws[0].upd_used = 0;
    CUDA_TRY(p, cudaEventRecord(p->ev[0], p->stream));
    if ((rc = upload_energies(p, energies, n_E, eta))) return rc;
    std::vector<double> hE(n_E);
    CUDA_TRY(p, cudaMemcpyAsync(hE.data(), p->E.p, sizeof(double) * (size_t)n_E, cudaMemcpyDeviceToHost, p->stream));
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    for (int k = 0; k < n_E; k++)
        if (!std::isfinite(hE[k])) return fail(p, RGF_EINVAL, "energies[%d] is not finite", k);
    const int batch = p->n_dev * n_E;
    int lead_open = 0;
    if ((rc = transmission_pass(p, n_E, eta, p->formulation, &lead_open))) return rc;
    int result = pass_result(p, n_E, lead_open, RGF_OK);
    if (result == RGF_ECUDA) return result;
    // ---- near-charge-neutrality guard of the half-slice formulation.  The cut between
    // B_i and F_i leaves the B atoms singly bonded; where their edge-like states are resonant the step loses
    // ~ 0.2 eps_mach (|t| max|gB|)^2.  The fused kernel records the smallest pivot of every matrix; items whose estimate
    // exceeds guard_tol are computed again in RGF_FORM_DENSE (no such cut) and replace the first result.
    p->guard_G.assign(batch, 0.0);
    p->guard_Gmax.assign(batch, 0.0);
    if (p->guard_tol > 0.0 && precision == RGF_C128 && use_fused(p)) {
        std::vector<unsigned> key(batch);
        std::vector<double> hT(batch), gsq(batch);
        CUDA_TRY(p, cudaMemcpyAsync(key.data(), p->pivmin.p, sizeof(unsigned) * (size_t)batch, cudaMemcpyDeviceToHost, p->stream));
        CUDA_TRY(p, cudaMemcpyAsync(gsq.data(), p->gsq.p, sizeof(double) * (size_t)batch, cudaMemcpyDeviceToHost, p->stream));
        CUDA_TRY(p, cudaMemcpyAsync(hT.data(), p->T.p, sizeof(double) * (size_t)batch, cudaMemcpyDeviceToHost, p->stream));
        CUDA_TRY(p, cudaStreamSynchronize(p->stream));
        std::vector<char> redo(n_E, 0);
        for (int b = 0; b < batch; b++) {
            const unsigned long long bits = ((unsigned long long)(key[b] << 8)) << 32;
            double piv;
            memcpy(&piv, &bits, sizeof(piv));
            p->guard_Gmax[b] = (key[b] == 0xffffffffu || !(piv > 0.0)) ? 0.0 : std::fabs(p->t) / piv;
            const double G = std::fabs(p->t) * std::sqrt(gsq[b] / (double)p->L);       // rms over the L B half-steps
            p->guard_G[b] = G;
            const double T = std::isfinite(hT[b]) ? std::fabs(hT[b]) : 1.0;
            if (!(kGuardC * G * G * T / std::max(1.0, T) <= p->guard_tol)) redo[b % n_E] = 1;
        }
        std::vector<int> idx;
        std::vector<double> E2;
        for (int e = 0; e < n_E; e++) if (redo[e]) { idx.push_back(e); E2.push_back(hE[e]); }
        const int n2 = (int)idx.size();
        p->stats.guard_redone = n2;
        if (n2 > 0) {
            if ((rc = ensure(p, p->T_keep, sizeof(double) * (size_t)batch))) return rc;
            if ((rc = ensure(p, p->redo_idx, sizeof(int) * (size_t)n2))) return rc;
            CUDA_TRY(p, cudaMemcpyAsync(p->T_keep.p, p->T.p, sizeof(double) * (size_t)batch, cudaMemcpyDeviceToDevice, p->stream));
            CUDA_TRY(p, cudaMemcpyAsync(p->redo_idx.p, idx.data(), sizeof(int) * (size_t)n2, cudaMemcpyHostToDevice, p->stream));
            CUDA_TRY(p, cudaMemcpyAsync(p->E.p, E2.data(), sizeof(double) * (size_t)n2, cudaMemcpyHostToDevice, p->stream));
            CUDA_TRY(p, cudaStreamSynchronize(p->stream));          // idx / E2 are host vectors
            int open2 = 0;
            if ((rc = transmission_pass(p, n2, eta, RGF_FORM_DENSE, &open2, false))) return rc;
            const int r2 = pass_result(p, n2, open2, RGF_OK);
            if (r2 != RGF_OK) result = r2;
            scatter_T_kernel<<<(p->n_dev * n2 + 255) / 256, 256, 0, p->stream>>>(ptr<double>(p->T_keep), ptr<double>(p->T), ptr<int>(p->redo_idx),
                                                                                n2, n_E, p->n_dev);
            p->stats.launches++;
            CUDA_TRY(p, cudaMemcpyAsync(p->T.p, p->T_keep.p, sizeof(double) * (size_t)batch, cudaMemcpyDeviceToDevice, p->stream));
            CUDA_TRY(p, cudaMemcpyAsync(p->E.p, hE.data(), sizeof(double) * (size_t)n_E, cudaMemcpyHostToDevice, p->stream));
            CUDA_TRY(p, cudaStreamSynchronize(p->stream));
        }
    }
    CUDA_TRY(p, cudaMemcpyAsync(T_out, p->T.p, sizeof(double) * (size_t)batch, cudaMemcpyDefault, p->stream));
    CUDA_TRY(p, cudaEventRecord(p->ev[4], p->stream));
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    drain_update_events(p);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, p->ev[0], p->ev[4]); p->stats.ms_total = ms;
    p->stats.ms_trace = p->stats.ms_total - p->stats.ms_leads - p->stats.ms_sweep;
    return result;
}

int rgf_destroy(rgf_plan *p)
{
    if (!p) return RGF_OK;
    cudaSetDevice(p->device);
    if (p->stream) cudaStreamSynchronize(p->stream);
    Buf *bufs[] = {&p->onsite, &p->bond, &p->hop, &p->bondc, &p->E, &p->T, &p->status, &p->lead_flags, &p->pivmin, &p->gsq, &p->T_keep, &p->redo_idx,
                   &p->gL, &p->gR, &p->l_eps, &p->l_eps_s, &p->l_alpha, &p->l_beta, &p->l_T1, &p->l_T2, &p->l_T3,
                   &p->l_W, &p->l_W2, &p->stage_in, &p->stage_out, &p->lc_S3, &p->lc_R, &p->lm_Q, &p->lead_status, &p->ld_A0, &p->ld_A1, &p->ld_B0, &p->ld_B1, &p->ld_stash, &p->ld_stashL, &p->ld_out};
    for (Buf *b : bufs) release(*b);
    for (Ws &w : p->ws) {
        if (w.stream) cudaStreamSynchronize(w.stream);
        Buf *wb[] = {&w.G0, &w.G1, &w.Nb, &w.rowAt, &w.orig, &w.Pa, &w.Pb, &w.H0, &w.H1, &w.H2, &w.Wc, &w.Tr, &w.Fx0, &w.Fx1, &w.Fp0, &w.Fp1, &w.Fperm, &w.Cp0, &w.Cp1};
        for (Buf *b : wb) release(*b);
        for (auto &pr : w.upd_events) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
        if (w.own_stream && w.stream) cudaStreamDestroy(w.stream);
    }
    for (int i = 0; i < 5; i++) if (p->ev[i]) cudaEventDestroy(p->ev[i]);
    for (int i = 0; i < 2; i++) if (p->ev_sync[i]) cudaEventDestroy(p->ev_sync[i]);
    for (Buf &b : p->jn) release(b);
    if (p->own_stream && p->stream) cudaStreamDestroy(p->stream);
    delete p;
    return RGF_OK;
}

const char *rgf_last_error(const rgf_plan *p) { return p ? p->err : kNoPlan; }

int rgf_get_stats(const rgf_plan *p, rgf_stats *out)
{
    if (!p || !out) return RGF_EINVAL;
    *out = p->stats;
    return RGF_OK;
}

int rgf_set_profiling(rgf_plan *p, int level)
{
    if (!p || level < 0 || level > 1) return RGF_EINVAL;
    p->profiling = level;
    return RGF_OK;
}

int rgf_set_formulation(rgf_plan *p, int formulation)
{
    if (!p || formulation < RGF_FORM_DENSE || formulation > RGF_FORM_HALF_STEPWISE) return RGF_EINVAL;
    p->formulation = formulation;
    return RGF_OK;
}

int rgf_set_lead_method(rgf_plan *p, int method)
{
    if (!p || method < RGF_LEAD_CELL_DENSE || method > RGF_LEAD_MODE_SPACE) return RGF_EINVAL;
    p->lead_method = method;
    return RGF_OK;
}

int rgf_set_guard(rgf_plan *p, double tol)
{
    if (!p || !(tol >= 0.0)) return RGF_EINVAL;
    p->guard_tol = tol;
    return RGF_OK;
}

int rgf_get_guard_indicators(const rgf_plan *p, double *Grms_out, double *Gmax_out, int n)
{
    if (!p || !Grms_out || n < 0) return RGF_EINVAL;
    for (int k = 0; k < n; k++) {
        Grms_out[k] = k < (int)p->guard_G.size() ? p->guard_G[k] : 0.0;
        if (Gmax_out) Gmax_out[k] = k < (int)p->guard_Gmax.size() ? p->guard_Gmax[k] : 0.0;
    }
    return RGF_OK;
}

int rgf_set_cohort(rgf_plan *p, int cohort)
{
    if (!p || cohort < 0) return RGF_EINVAL;
    p->cohort_override = cohort;
    return RGF_OK;
}

// FP64 tensor-pipe ceiling measured live: every warp issues independent DMMA.8x8x4 chains.
__global__ void fp64_peak_kernel(double *out, int iters)
{
    double a = threadIdx.x * 1e-3, b = threadIdx.x * 2e-3;
    double c[8][2];
#pragma unroll
    for (int j = 0; j < 8; j++) { c[j][0] = 0.0; c[j][1] = 0.0; }
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int j = 0; j < 8; j++) dmma884(c[j][0], c[j][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < 8; j++) s += c[j][0] + c[j][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

int rgf_fp64_peak_tflops(rgf_plan *p, double *tflops_out)
{
    int rc = begin_call(p);
    if (rc) return rc;
    if (!tflops_out) return fail(p, RGF_EINVAL, "tflops_out is NULL");
    int sms = 0;
    CUDA_TRY(p, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p->device));
    const int blocks = 2 * sms, threads = 512, iters = 40000;
    if ((rc = ensure(p, p->stage_out, sizeof(double) * (size_t)blocks * threads))) return rc;
    double best = 0.0;
    for (int rep = 0; rep < 4; rep++) {
        CUDA_TRY(p, cudaEventRecord(p->ev[0], p->stream));
        fp64_peak_kernel<<<blocks, threads, 0, p->stream>>>(ptr<double>(p->stage_out), iters);
        CUDA_TRY(p, cudaEventRecord(p->ev[1], p->stream));
        CUDA_TRY(p, cudaStreamSynchronize(p->stream));
        float ms = 0.f;
        CUDA_TRY(p, cudaEventElapsedTime(&ms, p->ev[0], p->ev[1]));
        double tf = (double)blocks * (threads / 32) * (double)iters * 8.0 * 512.0 / (ms * 1e-3) * 1e-12;
        if (rep > 0 && tf > best) best = tf;
    }
    *tflops_out = best;
    return RGF_OK;
}

int rgf_inverse_batched(rgf_plan *p, int n, int batch, const double *A, double *Ainv)
{
    int rc = begin_call(p);
    if (rc) return rc;
    if (n < 1 || batch < 1 || !A || !Ainv) return fail(p, RGF_EINVAL, "rgf_inverse_batched: bad argument");
    memset(&p->stats, 0, sizeof(p->stats));
    const size_t bytes = sizeof(cplx) * (size_t)n * n * batch;
    if ((rc = ensure(p, p->stage_in, bytes))) return rc;
    if ((rc = ensure(p, p->status, sizeof(int) * (size_t)batch))) return rc;
    if ((rc = ensure(p, p->stage_out, bytes))) return rc;
    if ((rc = ensure_inverse_ws(p, p->ws[0], n, batch))) return rc;
    CUDA_TRY(p, cudaMemcpyAsync(p->stage_in.p, A, bytes, cudaMemcpyDefault, p->stream));
    CUDA_TRY(p, cudaMemsetAsync(p->status.p, 0, sizeof(int) * (size_t)batch, p->stream));
    cplx *res = nullptr;
    if ((rc = run_inverse(p, p->ws[0], ptr<cplx>(p->stage_in), ptr<cplx>(p->stage_out), n, batch, ptr<int>(p->status), &res))) return rc;
    std::vector<int> h_status(batch);
    CUDA_TRY(p, cudaMemcpyAsync(Ainv, res, bytes, cudaMemcpyDefault, p->stream));
    CUDA_TRY(p, cudaMemcpyAsync(h_status.data(), p->status.p, sizeof(int) * (size_t)batch, cudaMemcpyDeviceToHost, p->stream));
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    drain_update_events(p);
    for (int b = 0; b < batch; b++)
        if (h_status[b]) return fail(p, RGF_ESINGULAR, "zero or non-finite pivot in matrix %d", b);
    return RGF_OK;
}

int rgf_lead_self_energy(rgf_plan *p, int dev, const double *energies, int n_E, double eta, int side, double *Sigma_out,
                         int *iterations_out)
{
    int rc = begin_call(p);
    if (rc) return rc;
    if (!p->has_device) return fail(p, RGF_ESTATE, "rgf_lead_self_energy before rgf_set_device");
    if (dev < 0 || dev >= p->n_dev || (side != 1 && side != -1) || !Sigma_out) return fail(p, RGF_EINVAL, "bad argument");
    memset(&p->stats, 0, sizeof(p->stats));
    if ((rc = upload_energies(p, energies, n_E, eta))) return rc;
    if ((rc = ensure(p, p->status, sizeof(int) * (size_t)n_E * p->n_dev))) return rc;
    CUDA_TRY(p, cudaMemsetAsync(p->status.p, 0, sizeof(int) * (size_t)n_E * p->n_dev, p->stream));
    int open = 0;
    if ((rc = run_leads(p, n_E, eta, &open))) return rc;
    const int M = p->M, L = p->L;
    const size_t MM = (size_t)M * M;
    const cplx *src = side < 0 ? ptr<cplx>(p->gL) : lead_gR(p);
    // Sigma = t^2 m (.) g (.) m, masked on the device (lead_sigma_kernel)
    if ((rc = ensure(p, p->stage_out, sizeof(cplx) * MM * n_E))) return rc;
    dim3 grid((unsigned)std::min<size_t>((MM + 255) / 256, 2048), n_E);
    lead_sigma_kernel<<<grid, 256, 0, p->stream>>>(ptr<cplx>(p->stage_out), src, ptr<uint8_t>(p->bond) + ((size_t)dev * (L + 1) + (side < 0 ? 0 : L)) * M, M, p->t);
    p->stats.launches++;
    CUDA_TRY(p, cudaGetLastError());
    CUDA_TRY(p, cudaMemcpyAsync(Sigma_out, p->stage_out.p, sizeof(cplx) * MM * n_E, cudaMemcpyDefault, p->stream));
    std::vector<int> h_ls(n_E);
    CUDA_TRY(p, cudaMemcpyAsync(h_ls.data(), p->lead_status.p, sizeof(int) * (size_t)n_E, cudaMemcpyDeviceToHost, p->stream));
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    for (int e = 0; e < n_E; e++)
        if (h_ls[e]) return fail(p, RGF_ESINGULAR, "zero or non-finite pivot in the lead decimation of energy %d", e);
    if (iterations_out) *iterations_out = p->stats.lead_iterations;
    if (open) return fail(p, RGF_ENOCONV, "lead decimation did not converge for %d energies", open);
    return RGF_OK;
}

int rgf_sweep_state(rgf_plan *p, int dev, const double *energies, int n_E, double eta, int precision, int nslices,
                    double *g_out, double *P_out)
{
    int rc = begin_call(p);
    if (rc) return rc;
    if (!p->has_device) return fail(p, RGF_ESTATE, "rgf_sweep_state before rgf_set_device");
    if (dev < 0 || dev >= p->n_dev || nslices < 1 || nslices > p->L || !g_out || !P_out) return fail(p, RGF_EINVAL, "bad argument");
    if (precision != RGF_C128 && precision != RGF_C64) return fail(p, RGF_EINVAL, "precision must be RGF_C128 or RGF_C64");
    if (precision == RGF_C64 && (p->formulation != RGF_FORM_HALF || p->nh > HC_NMAX))
        return fail(p, RGF_EUNSUPPORTED, "the complex64 sweep is built for RGF_FORM_HALF and M <= 256 only");
    p->precision = precision;
    memset(&p->stats, 0, sizeof(p->stats));
    if ((rc = upload_energies(p, energies, n_E, eta))) return rc;
    const int batch = p->n_dev * n_E, M = p->M, nh = p->nh;
    if ((rc = ensure(p, p->status, sizeof(int) * (size_t)batch))) return rc;
    CUDA_TRY(p, cudaMemsetAsync(p->status.p, 0, sizeof(int) * (size_t)batch, p->stream));
    if ((rc = ensure(p, p->pivmin, sizeof(unsigned) * (size_t)batch))) return rc;
    if ((rc = ensure(p, p->gsq, sizeof(double) * (size_t)batch))) return rc;
    if ((rc = run_leads(p, n_E, eta, nullptr))) return rc;
    Ws &w = p->ws[0];
    const bool half = p->formulation != RGF_FORM_DENSE;
    if ((rc = half ? ensure_sweep_ws_half(p, w, n_E) : ensure_sweep_ws(p, w, n_E))) return rc;
    cplx *G = nullptr, *Galt = nullptr, *Pcur = nullptr;
    const size_t bytes = sizeof(cplx) * (size_t)M * M * n_E;
    if ((rc = ensure(p, p->stage_out, bytes))) return rc;
    dim3 grid((unsigned)std::min((M * M + 255) / 256, 2048), n_E);
    if (half) {
        if ((rc = run_sweep_cohort_half(p, w, n_E, eta, dev * n_E, n_E, nslices, &G, &Pcur))) return rc;
        if ((rc = ensure(p, p->stage_in, bytes))) return rc;
        half_expand_g_kernel<<<grid, 256, 0, p->stream>>>(G, ptr<cplx>(p->stage_in), M, nh, (nslices - 1) & 1);
        G = ptr<cplx>(p->stage_in);
    } else {
        if ((rc = run_sweep_cohort(p, w, n_E, eta, dev * n_E, n_E, nslices, &G, &Galt, &Pcur))) return rc;
    }
    propagator_expand_kernel<<<grid, 256, 0, p->stream>>>(Pcur, ptr<cplx>(p->stage_out), M, nh, (nslices - 1) & 1);
    CUDA_TRY(p, cudaGetLastError());
    CUDA_TRY(p, cudaMemcpyAsync(g_out, G, bytes, cudaMemcpyDefault, p->stream));
    CUDA_TRY(p, cudaMemcpyAsync(P_out, p->stage_out.p, bytes, cudaMemcpyDefault, p->stream));
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    drain_update_events(p);
    return RGF_OK;
}

// ---- multi-GPU convention: (seed, energy) pairs are independent, so N ranks split the energy grid
// round-robin, rank r taking energies[r], energies[r + N], ...; no data-path collective.  Host-only helpers, no CUDA call.
int rgf_shard_count(int n_E, int world, int rank)
{
    if (n_E < 0 || world < 1 || rank < 0 || rank >= world) return RGF_EINVAL;
    return n_E > rank ? (n_E - rank + world - 1) / world : 0;
}

int rgf_shard_energies(const double *energies, int n_E, int world, int rank, double *shard_out)
{
    const int cnt = rgf_shard_count(n_E, world, rank);
    if (cnt < 0 || !energies || !shard_out) return RGF_EINVAL;
    for (int k = 0; k < cnt; k++) shard_out[k] = energies[rank + (long long)k * world];
    return cnt;
}

int rgf_unshard(const double *T_shard, int n_dev, int n_E, int world, int rank, double *T_full)
{
    const int cnt = rgf_shard_count(n_E, world, rank);
    if (cnt < 0 || n_dev < 1 || !T_shard || !T_full) return RGF_EINVAL;
    for (int d = 0; d < n_dev; d++)
        for (int k = 0; k < cnt; k++) T_full[(long long)d * n_E + rank + (long long)k * world] = T_shard[(long long)d * cnt + k];
    return RGF_OK;
}

// F-4: local density of states of the connected device, LDOS[n_dev][n_E][L][M] (ldos_kernels.cuh states the recursion).
// Three batched M x M inverses per slice and matrix: the gR chain and the gL chain run side by side on two streams and stash
// their (M/2)-blocks in HBM; the G_ii of all slices are then inverted in batches of (matrix, slice) pairs.  Matrices in
// chunks sized to at most half of the free memory.
int rgf_ldos(rgf_plan *p, const double *energies, int n_E, double eta, double *ldos_out)
{
    int rc = begin_call(p);
    if (rc) return rc;
    if (!p->has_device) return fail(p, RGF_ESTATE, "rgf_ldos before rgf_set_device");
    if (!ldos_out) return fail(p, RGF_EINVAL, "ldos_out is NULL");
    if (n_E >= 1 && (long long)p->n_dev * n_E > 65535)
        return fail(p, RGF_EUNSUPPORTED, "n_dev * n_E = %lld > 65535 batch items per call: split the energy grid", (long long)p->n_dev * n_E);
    memset(&p->stats, 0, sizeof(p->stats));
    CUDA_TRY(p, cudaEventRecord(p->ev[0], p->stream));
    if ((rc = upload_energies(p, energies, n_E, eta))) return rc;
    const int M = p->M, L = p->L, nh = p->nh, batch = p->n_dev * n_E;
    const size_t MM = (size_t)M * M;
    if ((rc = ensure(p, p->status, sizeof(int) * (size_t)batch))) return rc;
    CUDA_TRY(p, cudaMemsetAsync(p->status.p, 0, sizeof(int) * (size_t)batch, p->stream));
    int lead_open = 0;
    if ((rc = run_leads(p, n_E, eta, &lead_open))) return rc;
    if (lead_open) return fail(p, RGF_ENOCONV, "lead decimation did not converge for %d energies", lead_open);
    // chunk of matrices whose two stashes fit
    size_t free_b = 0, total_b = 0;
    CUDA_TRY(p, cudaMemGetInfo(&free_b, &total_b));
    Ws &wl = p->ws[0], &wr = p->ws[1];
    const size_t per_matrix = sizeof(cplx) * (2 * (size_t)L * nh * nh + 4 * MM) + sizeof(double) * (size_t)L * M + sizeof(cplx) * (size_t)M * 256;
    const size_t held = p->ld_stash.cap + p->ld_stashL.cap + p->ld_out.cap + p->ld_A0.cap + p->ld_A1.cap + wl.G0.cap + wl.G1.cap + wr.G0.cap + wr.G1.cap;
    const size_t have = free_b / 2 + held;
    int chunk = (int)std::min<size_t>((size_t)batch, std::max<size_t>(1, have / per_matrix));
    if ((rc = ensure_sweep_ws(p, wl, chunk)) || (rc = ensure_sweep_ws(p, wr, chunk))) return rc;
    if ((rc = ensure(p, p->ld_stash, sizeof(cplx) * (size_t)L * nh * nh * chunk))) return rc;
    if ((rc = ensure(p, p->ld_stashL, sizeof(cplx) * (size_t)L * nh * nh * chunk))) return rc;
    if ((rc = ensure(p, p->ld_out, sizeof(double) * (size_t)L * M * chunk))) return rc;
    // batches of (matrix, slice) pairs for the G_ii: about 2048 matrices at a time
    const int ns_max = std::max(1, std::min(L, 2048 / std::max(1, chunk)));
    const int bmax = ns_max * chunk;
    if ((rc = ensure(p, p->ld_A0, sizeof(cplx) * MM * bmax)) || (rc = ensure(p, p->ld_A1, sizeof(cplx) * MM * bmax))) return rc;
    if ((rc = ensure(p, p->ld_B0, sizeof(int) * (size_t)bmax))) return rc;
    if ((rc = ensure_inverse_ws(p, wl, M, bmax))) return rc;
    p->stats.cohort = chunk;
    const double *E = ptr<double>(p->E);
    const cplx *gLl = ptr<cplx>(p->gL), *gRl = lead_gR(p);
    cplx *stashR = ptr<cplx>(p->ld_stash), *stashL = ptr<cplx>(p->ld_stashL);
    for (int bz0 = 0; bz0 < batch; bz0 += chunk) {
        const int nb = std::min(chunk, batch - bz0);
        int *status = ptr<int>(p->status) + bz0;
        dim3 ag((unsigned)std::min<size_t>((MM + 255) / 256, 2048), nb), sg((unsigned)std::min((nh * nh + 255) / 256, 1024), nb);
        const size_t sslice = (size_t)nh * nh * nb;          // stash of one slice for the chunk
        // ---- the two chains side by side: gR_i (i = L-1 .. 1) on the second stream, gL_i (i = 0 .. L-2) on the plan's
        CUDA_TRY(p, cudaEventRecord(p->ev_sync[0], p->stream));
        CUDA_TRY(p, cudaStreamWaitEvent(wr.stream, p->ev_sync[0], 0));
        cplx *RA = ptr<cplx>(wr.G0), *RB = ptr<cplx>(wr.G1), *LA = ptr<cplx>(wl.G0), *LB = ptr<cplx>(wl.G1), *Lprev = nullptr, *res = nullptr;
        for (int s = 0; s < L - 1; s++) {
            {   // right chain, slice i: A from the stashed block of gR_{i+1} (or the lead)
                const int i = L - 1 - s;
                ldos_assemble_kernel<<<ag, 256, 0, wr.stream>>>(RA, M, L, nh, i, n_E, bz0, E, eta, p->t, ptr<double>(p->onsite), ptr<uint8_t>(p->bond),
                                                               ptr<uint8_t>(p->hop), 0, nullptr, gLl, 1, i + 1 < L ? stashR + (size_t)(i + 1) * sslice : nullptr, gRl);
                if ((rc = run_inverse(p, wr, RA, RB, M, nb, status, &res))) return rc;
                ldos_stash_kernel<<<sg, 256, 0, wr.stream>>>(res, stashR + (size_t)i * sslice, M, nh, (i - 1) & 1);
                p->stats.launches += 2;
            }
            {   // left chain, slice i: A from the full gL_{i-1} of the previous step (or the lead)
                const int i = s;
                cplx *dst = (Lprev == LA) ? LB : LA;
                ldos_assemble_kernel<<<ag, 256, 0, wl.stream>>>(dst, M, L, nh, i, n_E, bz0, E, eta, p->t, ptr<double>(p->onsite), ptr<uint8_t>(p->bond),
                                                               ptr<uint8_t>(p->hop), 1, Lprev, gLl, 0, nullptr, gRl);
                if ((rc = run_inverse(p, wl, dst, dst == LA ? LB : LA, M, nb, status, &res))) return rc;
                Lprev = res;
                ldos_stash_kernel<<<sg, 256, 0, wl.stream>>>(res, stashL + (size_t)i * sslice, M, nh, i & 1);
                p->stats.launches += 2;
            }
        }
        CUDA_TRY(p, cudaGetLastError());
        CUDA_TRY(p, cudaEventRecord(p->ev_sync[1], wr.stream));
        CUDA_TRY(p, cudaStreamWaitEvent(p->stream, p->ev_sync[1], 0));
        // ---- G_ii of all slices: independent, in batches of ns slices x nb matrices
        int *dstat = ptr<int>(p->ld_B0);
        for (int i0 = 0; i0 < L; i0 += ns_max) {
            const int ns = std::min(ns_max, L - i0), nbat = ns * nb;
            dim3 bg((unsigned)std::min<size_t>((MM + 255) / 256, 64), nbat);
            ldos_assemble_both_kernel<<<bg, 256, 0, p->stream>>>(ptr<cplx>(p->ld_A0), M, L, nh, i0, nb, n_E, bz0, E, eta, p->t, ptr<double>(p->onsite),
                                                                ptr<uint8_t>(p->bond), ptr<uint8_t>(p->hop), stashL, stashR, gLl, gRl);
            CUDA_TRY(p, cudaMemsetAsync(dstat, 0, sizeof(int) * (size_t)nbat, p->stream));
            if ((rc = run_inverse(p, wl, ptr<cplx>(p->ld_A0), ptr<cplx>(p->ld_A1), M, nbat, dstat, &res))) return rc;
            const long long tot = (long long)nbat * M;
            ldos_diag_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, p->stream>>>(res, ptr<double>(p->ld_out), dstat, status, M, L, i0, nb, ns);
            p->stats.launches += 2;
        }
        CUDA_TRY(p, cudaGetLastError());
        CUDA_TRY(p, cudaMemcpyAsync(ldos_out + (size_t)bz0 * L * M, p->ld_out.p, sizeof(double) * (size_t)L * M * nb, cudaMemcpyDefault, p->stream));
        CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    }
    CUDA_TRY(p, cudaEventRecord(p->ev[4], p->stream));
    std::vector<int> h_status(batch);
    CUDA_TRY(p, cudaMemcpyAsync(h_status.data(), p->status.p, sizeof(int) * (size_t)batch, cudaMemcpyDeviceToHost, p->stream));
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    drain_update_events(p);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, p->ev[0], p->ev[4]); p->stats.ms_total = ms; p->stats.ms_sweep = ms;
    for (int b = 0; b < batch; b++)
        if (h_status[b]) return fail(p, RGF_ESINGULAR, "zero or non-finite pivot (first at batch item %d); its LDOS is NaN from that slice on", b);
    return RGF_OK;
}

}  // extern "C"

// ==========================================================================================
// Allocation-free entry point: rgf_inverse_batched_static (include/rgf.h).  A4 alone -- the n <= 256 path of
// run_inverse (gj32_panel_kernel / gj32_update_kernel / gj32_unpermute_kernel, the same kernels) -- with every byte of
// scratch in ONE file-scope device array, for callers that cannot call cudaMalloc (CUDA graph capture, tight serving
// loops, harnesses that forbid it).  It takes no plan (a plan owns streams, events and buffers) and calls no cudaMalloc /
// cudaFree / allocating library routine.  Every GPU that loads the library holds the array until exit.
// ==========================================================================================
#define RGF_STATIC_SCRATCH_BYTES (2ull * RGF_STATIC_MAX_ELEMS * 16 + (unsigned long long)RGF_STATIC_MAX_BATCH * 64 * 32 * 16 \
                                  + 2ull * RGF_STATIC_MAX_BATCH * 64 * 4 + 4096)
static __device__ __align__(256) unsigned char rgf_static_scratch[RGF_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kStaticMaxDevices = 64;
struct StaticSetup { bool done; unsigned char *base; };
StaticSetup g_static[kStaticMaxDevices];
thread_local char g_static_err[256] = "";

int static_fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_static_err, sizeof(g_static_err), fmt, ap);
    va_end(ap);
    return code;
}

// once per device, with that device current: the DEVICE address of the scratch array (in host code the array's name is
// only a stand-in) and the shared-memory attributes of the two kernels that need more than 48 KB
int static_setup(int dev, unsigned char **base)
{
    static std::mutex mu;
    std::lock_guard<std::mutex> lock(mu);
    if (!g_static[dev].done) {
        void *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, rgf_static_scratch);
        if (e != cudaSuccess || !ptr) return static_fail(RGF_ECUDA, "cudaGetSymbolAddress(rgf_static_scratch) failed on device %d: %s", dev, cudaGetErrorString(e));
        if ((e = cudaFuncSetAttribute(gj32_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gj32_panel_smem(256))) != cudaSuccess ||
            (e = cudaFuncSetAttribute(gj32_update_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GU32_SMEM)) != cudaSuccess)
            return static_fail(RGF_ECUDA, "cudaFuncSetAttribute failed on device %d: %s", dev, cudaGetErrorString(e));
        g_static[dev].base = static_cast<unsigned char *>(ptr);
        g_static[dev].done = true;
    }
    *base = g_static[dev].base;
    return RGF_OK;
}

bool is_device_pointer(const void *p, int dev)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) && at.device == dev;
}

}  // namespace

extern "C" {

const char *rgf_static_last_error(void) { return g_static_err; }

int rgf_inverse_batched_static(int cuda_device, void *cuda_stream, int n, int batch, const double *A_dev, double *Ainv_dev, int *status_dev)
{
    g_static_err[0] = 0;
    if (n < 1 || batch < 1 || !A_dev || !Ainv_dev) return static_fail(RGF_EINVAL, "rgf_inverse_batched_static: need n >= 1, batch >= 1, A_dev and Ainv_dev non-NULL");
    if (n > RGF_STATIC_MAX_N || batch > RGF_STATIC_MAX_BATCH || (long long)n * n * batch > RGF_STATIC_MAX_ELEMS || (long long)n * batch > 64LL * RGF_STATIC_MAX_BATCH)
        return static_fail(RGF_EUNSUPPORTED, "rgf_inverse_batched_static: n = %d, batch = %d exceeds the static scratch (n <= %d, batch <= %d, n*n*batch <= %d, n*batch <= %d); "
                           "use rgf_inverse_batched", n, batch, RGF_STATIC_MAX_N, RGF_STATIC_MAX_BATCH, RGF_STATIC_MAX_ELEMS, 64 * RGF_STATIC_MAX_BATCH);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev || cuda_device >= kStaticMaxDevices)
        return static_fail(RGF_ECUDA, "rgf_inverse_batched_static: no CUDA device %d", cuda_device);
    cudaError_t e;
    if ((e = cudaSetDevice(cuda_device)) != cudaSuccess) return static_fail(RGF_ECUDA, "cudaSetDevice(%d): %s", cuda_device, cudaGetErrorString(e));
    if (!is_device_pointer(A_dev, cuda_device) || !is_device_pointer(Ainv_dev, cuda_device) || (status_dev && !is_device_pointer(status_dev, cuda_device)))
        return static_fail(RGF_EINVAL, "rgf_inverse_batched_static: A_dev, Ainv_dev and status_dev must be device pointers on device %d", cuda_device);
    unsigned char *base = nullptr;
    int rc = static_setup(cuda_device, &base);
    if (rc) return rc;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    // carve the array: two n x n work buffers per matrix, the multipliers of a panel, the two row maps, the flags
    const long long gb = (long long)n * n;
    cplx *X = reinterpret_cast<cplx *>(base);
    cplx *Y = X + RGF_STATIC_MAX_ELEMS;
    cplx *Mult = Y + RGF_STATIC_MAX_ELEMS;
    int *rowAt = reinterpret_cast<int *>(Mult + (size_t)RGF_STATIC_MAX_BATCH * 64 * 32);
    int *orig = rowAt + RGF_STATIC_MAX_BATCH * 64;
    int *status = orig + RGF_STATIC_MAX_BATCH * 64;
    // the array keeps the last call's contents: the flags must start at zero, orig at the identity; X, Mult, rowAt are
    // fully written before they are read, Y only ever holds what this call's panels and updates wrote
    if ((e = cudaMemsetAsync(status, 0, sizeof(int) * (size_t)batch, stream)) != cudaSuccess ||
        (e = cudaMemcpyAsync(X, A_dev, sizeof(cplx) * (size_t)gb * batch, cudaMemcpyDeviceToDevice, stream)) != cudaSuccess)
        return static_fail(RGF_ECUDA, "rgf_inverse_batched_static: %s", cudaGetErrorString(e));
    const int total = n * batch;
    gj_init_orig_kernel<<<(total + 255) / 256, 256, 0, stream>>>(orig, n, total);
    for (int k0 = 0; k0 < n; k0 += G32_B) {
        gj32_panel_kernel<<<batch, G32_NT, gj32_panel_smem(n), stream>>>(X, Y, gb, n, k0, Mult, rowAt, orig, status);
        if (n > G32_B) {
            dim3 grid((n + GU32_BN - 1) / GU32_BN, (n + GU32_BM - 1) / GU32_BM, batch);
            gj32_update_kernel<<<grid, GU32_THREADS, GU32_SMEM, stream>>>(X, Y, gb, n, k0, Mult, rowAt);
        }
        std::swap(X, Y);
    }
    dim3 grid((n + 7) / 8, batch);
    gj32_unpermute_kernel<<<grid, 256, 0, stream>>>(X, reinterpret_cast<cplx *>(Ainv_dev), gb, n, orig);
    if (status_dev && (e = cudaMemcpyAsync(status_dev, status, sizeof(int) * (size_t)batch, cudaMemcpyDeviceToDevice, stream)) != cudaSuccess)
        return static_fail(RGF_ECUDA, "rgf_inverse_batched_static: %s", cudaGetErrorString(e));
    if ((e = cudaGetLastError()) != cudaSuccess) return static_fail(RGF_ECUDA, "rgf_inverse_batched_static: launch failed: %s", cudaGetErrorString(e));
    return RGF_OK;
}

}  // extern "C"
