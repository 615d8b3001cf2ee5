/*
 * rgf.h -- C ABI of the B200 (sm_100a) recursive Green's function library.
 *
 * What the library computes: the Landauer transmission T(E) of an armchair graphene
 * nanoribbon (one p_z orbital per atom, nearest-neighbour hopping t) between two clean
 * semi-infinite leads of the same width, by the recursive Green's function sweep of
 *   S. Ihnatsenka, Comput. Phys. Commun. 183 (2012) 543 (arXiv:1107.5300):
 *     PAPER.md:33-37  Eq. 1   G = (E - H)^-1
 *     PAPER.md:37-41  Eq. 2   conductance = (2e^2/h) Tr[Gamma_L G^a Gamma_R G^r]
 *     PAPER.md:45-53  Eq. 4-5 slice recursion  G_jj, G_1j  (one solver call + GEMMs per slice)
 *     PAPER.md:53,58  lead self-energies added at the first and the last slice
 * in the direct form of BASELINE.json:north_star, with z = E + i*eta:
 *     G_ii   = (z - H_i - V G_{i-1,i-1} V)^-1            (complex M x M inverse)
 *     G_{i,0} = G_ii V G_{i-1,0}                           (complex GEMM)
 *     Sigma_L/R from Sancho-Rubio decimation of the clean two-slice lead cell
 *     T(E) = Re Tr[Gamma_L G_{L-1,0}^dagger Gamma_R G_{L-1,0}],  Gamma = i(Sigma - Sigma^dagger)
 *
 * Geometry (BASELINE.json:configs[0]): M atoms per slice (matrix size),
 * L slices, 0-based slice i and atom j.  H_i = diag(onsite[i][:]) + t on the first sub/super
 * diagonal; V_{i,i+1} = t*diag(m_i), m_i[j] = 1 iff (i+j) even.  A vacancy zeroes every
 * hopping that touches the site (it stays an isolated level at its on-site energy).
 *
 * Every step runs in CUDA kernels of this library; there is no CPU fallback.  All entry
 * points return RGF_OK (0) or a negative error code, never throw, never abort.
 *
 * Pointers: unless stated otherwise an array argument may be a HOST pointer or a CUDA DEVICE
 * pointer on the plan's device (the library asks cudaPointerGetAttributes); the caller owns
 * every array, and the library never keeps a caller pointer after the call returns.
 */
#ifndef RGF_H
#define RGF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rgf_plan rgf_plan;          /* opaque; created by rgf_plan_create, freed by rgf_destroy */

enum { RGF_C128 = 0, RGF_C64 = 1 };        /* precision of the sweep (assembly, inverse, propagator) */

enum {
    RGF_OK = 0,
    RGF_EINVAL = -1,       /* bad argument (NULL, M < 2, L < 1, n_E < 1, eta <= 0, non-finite, ...) */
    RGF_ECUDA = -2,        /* a CUDA call failed; see rgf_last_error                              */
    RGF_ENOMEM = -3,       /* host or device allocation failed                                    */
    RGF_ENOCONV = -4,      /* lead decimation hit the iteration cap for at least one energy       */
    RGF_ESINGULAR = -5,    /* zero or non-finite pivot in at least one inverse                    */
    RGF_ESTATE = -6,       /* rgf_transmission before rgf_set_device                              */
    RGF_EUNSUPPORTED = -7  /* precision / size not built in this version                          */
};

/* Create an empty plan bound to CUDA device `cuda_device`.  `cuda_stream` is a cudaStream_t
 * (e.g. torch.cuda.current_stream().cuda_stream) on which all work is enqueued, or NULL for a
 * stream owned by the plan.  *out receives the plan. */
int rgf_plan_create(rgf_plan **out, int cuda_device, void *cuda_stream);

/* Describe one ribbon (region of length L between two leads of the same width).
 *   onsite  [L][M] row-major doubles, eV
 *   t       hopping, eV (e.g. -2.7)
 *   vacancy [L][M] bytes, 1 = vacant site, or NULL for none
 * The arrays are copied to the device; the caller may free them on return.  A second call
 * replaces the device (buffers are reused when M and L are unchanged). */
int rgf_set_device(rgf_plan *p, int M, int L, const double *onsite, double t, const uint8_t *vacancy);

/* Batched variant: n_dev ribbons (disorder seeds) of the same M, L, t
 * (BASELINE.json:configs[1] "4 disorder seeds batched").  onsite [n_dev][L][M],
 * vacancy [n_dev][L][M] or NULL.  rgf_transmission then writes T_out[n_dev][n_E]. */
int rgf_set_device_batch(rgf_plan *p, int n_dev, int M, int L, const double *onsite, double t,
                         const uint8_t *vacancy);

/* T(E) for n_E energies (eV), broadening eta > 0 (eV), sweep precision RGF_C128 / RGF_C64.
 * T_out[n_dev][n_E] doubles (n_dev = 1 after rgf_set_device; n_dev * n_E <= 65535 per call).  Synchronous: T_out is valid on
 * return.  Runs leads (A2), the sweep (A3-A5) and the trace (A6) on the GPU.  On a per-energy
 * failure that entry of T_out is NaN, the other energies are still computed, and the code
 * (RGF_ENOCONV / RGF_ESINGULAR) is returned. */
int rgf_transmission(rgf_plan *p, const double *energies, int n_E, double eta, int precision,
                     double *T_out);

/* Free the plan and everything it owns.  NULL is accepted. */
int rgf_destroy(rgf_plan *p);

/* Message of the last error on this plan (plan-owned, valid until the next call), or a static
 * string if p is NULL. */
const char *rgf_last_error(const rgf_plan *p);

/* ---- counters of the last rgf_transmission call -------------------------------------- */
typedef struct rgf_stats {
    double ms_total;            /* CUDA-event time of the whole call on the plan's stream       */
    double ms_leads;            /* lead decimation                                               */
    double ms_sweep;            /* assembly + inverse + propagator over all slices              */
    double ms_trace;            /* Gamma trace + download                                        */
    double ms_inverse_update;   /* summed CUDA-event time of the dominant kernel of the sweep: the fused
                                   half_sweep_kernel (RGF_FORM_HALF, M <= 256), else the Gauss-Jordan update   */
    long long launches;         /* kernels launched by the call                                  */
    long long launches_inverse_update; /* launches of that kernel in the sweep (the ones timed)       */
    long long launches_leads;   /* kernels launched by the lead decimation                       */
    int lead_iterations;        /* decimation iterations run (max over energies)                 */
    int cohort;                 /* matrices per launch                                           */
    int guard_redone;           /* energies recomputed in RGF_FORM_DENSE by the near-neutrality guard */
    int reserved;
    double ms_guard;            /* of ms_total: the guard's second pass (leads + dense sweep + trace of the redone energies) */
} rgf_stats;
int rgf_get_stats(const rgf_plan *p, rgf_stats *out);

/* Timing detail: 0 = whole-call events only (default), 1 = also bracket every inverse-update
 * launch with events (adds a little launch overhead; used by bench.py for the roofline line). */
int rgf_set_profiling(rgf_plan *p, int level);

/* Formulation of the sweep.  Both are the recursion of PAPER.md:47-51 (Eq. 4-5) and give the same T(E):
 *   RGF_FORM_DENSE  one step per slice: complex M x M inverse + compact propagator GEMM, as
 *                   BASELINE.json:north_star words it (8 M^3 + M^3 real flops per slice-step);
 *   RGF_FORM_HALF   (default) the same recursion on the finer slicing B_0, F_0, B_1, F_1, ... where
 *                   F_i / B_i are the atoms of slice i bonded forwards / backwards (the armchair
 *                   inter-slice coupling t*diag(mask) touches only one of them): two steps per slice,
 *                   each a complex (M/2) x (M/2) inverse + (M/2)^3 GEMM (4 M^3 real flops per slice-step).
 *                   For M <= 256 the whole sweep of one (device, energy) pair is ONE fused kernel
 *                   (one CTA per pair; inverse and propagator product are a single Gauss-Jordan
 *                   elimination on [A | C P]); larger M runs it operation by operation;
 *   RGF_FORM_HALF_STEPWISE  the half-slice recursion launched operation by operation for every M
 *                   (what RGF_FORM_HALF does for M > 256; exported so that it is testable at small M).
 * In the half-slice formulations rgf_sweep_state returns only the F_i x F_i block of G_ii (NaN elsewhere). */
enum { RGF_FORM_DENSE = 0, RGF_FORM_HALF = 1, RGF_FORM_HALF_STEPWISE = 2 };
int rgf_set_formulation(rgf_plan *p, int formulation);

/* How the lead surface Green's functions (A2) are computed.  All three give the same Sigma_L/R (tested against the oracle):
 *   RGF_LEAD_MODE_SPACE  (default) the paper's own route ("solution of an eigen-problem"): in the transverse
 *                        sine basis the clean armchair lead decouples into M/2 chains with alternating hoppings
 *                        2t cos(p pi/(M+1)) and t; the surface Green's function of each chain is a closed form (root of a
 *                        quadratic), transformed back by one real x complex product per energy.  O(M) + one product,
 *                        no iteration, no host synchronisation, no resonance of the isolated cell;
 *   RGF_LEAD_CELL_DENSE  Sancho-Rubio decimation of the two-slice cell (BASELINE.json:north_star item 4) with one pivoted
 *                        2M x 2M inverse per iteration + 8 products of size M;
 *   RGF_LEAD_CELL_SCHUR  the same decimation on the (M/2)-blocks alpha, beta and the corrections really occupy; the corner
 *                        blocks of the cell's inverse come from one pivoted inverse of the M x M Schur complement on the
 *                        atoms that bond to the neighbouring cells: 8x fewer flops.  Falls back to RGF_LEAD_CELL_DENSE for
 *                        a call with an energy within 1 % of +-t, where the closed elimination is resonant. */
enum { RGF_LEAD_CELL_DENSE = 0, RGF_LEAD_CELL_SCHUR = 1, RGF_LEAD_MODE_SPACE = 2 };
int rgf_set_lead_method(rgf_plan *p, int method);

/* Near-charge-neutrality guard of RGF_FORM_HALF (complex128, fused kernel).  The cut between the two halves of a slice
 * leaves singly bonded atoms whose edge-like states are resonant close to charge neutrality (PAPER.md:82 is about
 * exactly this energy range); a B half-step with smallest pivot p loses about eps_mach (|t| / p)^2.  The fused
 * kernel records that pivot for every B half-step of every (device, energy) pair; with G the root mean square of
 * |t| / p over the L B half-steps (in a clean ribbon every half-step has the same p), every energy with
 *     1.5e-16 G^2 min(1, T) > tol
 * for some device is computed again in RGF_FORM_DENSE, which has no such cut, inside the same rgf_transmission call
 * (the constant is calibrated in DESIGN.md section 1a).  tol = 0 switches the guard off; default 1e-10, a tenth of the
 * tolerance 1e-9 max(1, T).  rgf_stats.guard_redone counts the energies recomputed. */
int rgf_set_guard(rgf_plan *p, double tol);
/* Indicators of the first pass of the last rgf_transmission call, [n_dev][n_E] each (HOST pointers; 0 where not
 * recorded): Grms_out = G above, Gmax_out (may be NULL) = |t| / (smallest pivot of the whole sweep). */
int rgf_get_guard_indicators(const rgf_plan *p, double *Grms_out, double *Gmax_out, int n);

/* Matrices per kernel launch in the sweep (0 = library default).  RGF_FORM_DENSE / _STEPWISE and the complex64 sweep:
 * the sweep runs cohort after cohort over all slices.  RGF_FORM_HALF in complex128 (fused kernel): the whole batch is one
 * cohort and `cohort` bounds the units (matrix, 64 half-steps) per launch instead, default = the number of resident CTA
 * slots of the GPU; with fewer slots than matrices every matrix is resumed from the state it left in HBM. */
int rgf_set_cohort(rgf_plan *p, int cohort);

/* Measures the FP64 tensor-pipe ceiling of the plan's GPU (independent DMMA.8x8x4 chains on every
 * warp, 2 CTAs x 16 warps per SM) and writes it in TFLOP/s; the roofline denominator of bench.py. */
int rgf_fp64_peak_tflops(rgf_plan *p, double *tflops_out);

/* ---- sub-steps, exported so that each row of the hot path can be checked on its own ---- */

/* A4 alone: inverse of `batch` complex n x n matrices (interleaved re,im doubles, row-major,
 * matrix b at A + b*n*n*2 doubles) by the library's blocked Gauss-Jordan with partial
 * pivoting.  A and Ainv may be host or device pointers; Ainv may equal A. */
int rgf_inverse_batched(rgf_plan *p, int n, int batch, const double *A, double *Ainv);

/* A2 alone: lead self-energies Sigma_L (side = -1) or Sigma_R (side = +1) of device `dev`
 * for n_E energies: Sigma_out[n_E][M][M] interleaved complex.  iterations_out (host int, may be
 * NULL) receives the number of decimation iterations run. */
int rgf_lead_self_energy(rgf_plan *p, int dev, const double *energies, int n_E, double eta, int side,
                         double *Sigma_out, int *iterations_out);

/* A3-A5 alone: state after the first `nslices` slices (1..L) of the sweep on device `dev`:
 * g_out[n_E][M][M] = G_ii and P_out[n_E][M][M] = G_{i,0}, i = nslices-1 (interleaved complex).
 * The library propagates only the rows/columns of G_{i,0} that the rest of the path consumes
 * (rows with m_i = 1, columns with m_{-1} = 1); every other entry of P_out is written as NaN. */
int rgf_sweep_state(rgf_plan *p, int dev, const double *energies, int n_E, double eta, int precision,
                    int nslices, double *g_out, double *P_out);

/* ---- multi-GPU convention (the path shards over energies, nothing is exchanged) -------------------------
 * One process per GPU, each with its own plan; rank r of `world` computes energies[r], energies[r + world], ... (round-robin:
 * the cost per energy is uniform but failures and guard redos cluster near charge neutrality).  HOST pointers only.
 *   rgf_shard_count     number of energies of rank `rank` (or RGF_EINVAL)
 *   rgf_shard_energies  writes them to shard_out[count]; returns count
 *   rgf_unshard         scatters a rank's result T_shard[n_dev][count] into its places of T_full[n_dev][n_E]; after every
 *                       rank's part has been scattered (e.g. from an all-gather) T_full is the single-GPU result. */
int rgf_shard_count(int n_E, int world, int rank);
int rgf_shard_energies(const double *energies, int n_E, int world, int rank, double *shard_out);
int rgf_unshard(const double *T_shard, int n_dev, int n_E, int world, int rank, double *T_full);

/* ---- second workload on the same kernels ---------------------------------------------------------
 * Local density of states of the device connected to both leads ("any desired quantity, e.g. charge density";
 * the Green's functions of the whole region):
 *     ldos_out[n_dev][n_E][L][M] = -(1/pi) Im G_ii[j][j],   G = (z - H_device - Sigma_L (+) 0 (+) Sigma_R)^-1  (Eq. 1)
 * by the recursion applied from both ends (three batched M x M inverses per slice; only the (M/2)-blocks the inter-slice
 * coupling keeps are stored between the two passes, in chunks of matrices that fit half of the free device memory).
 * The charge density is the caller's energy integral of it.  energies / ldos_out: host or device pointers; complex128;
 * eta as in rgf_transmission (an LDOS on a grid wants eta of the order of the grid spacing).  A matrix that hits a zero /
 * non-finite pivot has NaN from that slice on and RGF_ESINGULAR is returned. */
int rgf_ldos(rgf_plan *p, const double *energies, int n_E, double eta, double *ldos_out);

/* ---- allocation-free entry point --------------------------------------------------------------------------
 * A4 alone like rgf_inverse_batched (same kernels, n <= 256 path), for callers that cannot call cudaMalloc: code under CUDA
 * graph capture, tight serving loops, harnesses that forbid allocation.  It takes no plan and calls no cudaMalloc, cudaFree
 * or other allocating routine: all scratch (two work copies of the batch, the panel multipliers, the row maps, the pivot
 * flags) lives in one file-scope __device__ array of RGF_STATIC_SCRATCH_MB that every GPU loading the library holds until exit.
 *   cuda_device / cuda_stream   device ordinal and cudaStream_t (NULL = default stream) the work is enqueued on
 *   A_dev, Ainv_dev             DEVICE pointers on that device: batch complex n x n matrices, interleaved re,im doubles,
 *                               row-major, matrix b at + b*n*n*2 doubles.  A_dev is not modified; Ainv_dev may equal A_dev.
 *   status_dev                  DEVICE pointer to batch ints or NULL: 1 where a pivot was zero / non-finite, else 0.
 * Asynchronous: results are valid once the stream has completed the call.  Limits: n <= RGF_STATIC_MAX_N,
 * batch <= RGF_STATIC_MAX_BATCH, n*n*batch <= RGF_STATIC_MAX_ELEMS, n*batch <= 64*RGF_STATIC_MAX_BATCH; anything larger
 * returns RGF_EUNSUPPORTED (message: rgf_static_last_error) -- use rgf_inverse_batched.  Host pointers return RGF_EINVAL.
 * Every call on a device shares the one array, which keeps the last call's contents (the call clears what must start
 * at zero): two calls that overlap on the GPU -- different streams, or two host threads -- RACE; serialise them on one
 * stream or with events.  The array's address is resolved once per device (cudaGetSymbolAddress with that device current). */
#define RGF_STATIC_MAX_N 256
#define RGF_STATIC_MAX_BATCH 64
#define RGF_STATIC_MAX_ELEMS 262144
#define RGF_STATIC_SCRATCH_MB 10.04
int rgf_inverse_batched_static(int cuda_device, void *cuda_stream, int n, int batch, const double *A_dev, double *Ainv_dev,
                               int *status_dev);
const char *rgf_static_last_error(void);     /* message of the last failed rgf_inverse_batched_static call of this thread */

#ifdef __cplusplus
}
#endif
#endif /* RGF_H */
