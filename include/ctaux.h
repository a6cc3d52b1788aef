/* ctaux.h -- C ABI of the B200-native CT-AUX walker (libctaux_b200.so).
 *
 * The library runs the hot path of the continuous-time auxiliary-field QMC cluster solver of
 * DCA++ (arXiv:1901.01047, section 2.3) for B independent Markov chains
 * ("walkers") on ONE sm_100a device:
 *
 *   S1  G0 interpolation and construction of A_sigma = N_sigma^{-1}
 *       (Eq. (27); BASELINE.json: N^-1 = e^{-gamma sigma V} - G0 (e^{-gamma sigma V} - 1))
 *   S2  candidate products for the determinant ratios of a block of proposals
 *   S3  Metropolis proposals (vertex insertion / removal) evaluated over the small
 *       delayed block (submatrix updates)
 *   S4  the delayed rank-r flush  N <- N - U S^{-1} V^T  as FP64 tensor-core (DMMA) GEMMs
 *   S5  from-scratch rebuild  N = A^{-1}  by LU with partial pivoting
 *
 * Conventions (every reading of a point the paper leaves open is listed in DESIGN.md):
 *   - No torch types, no C++ types, no exceptions cross this boundary.
 *   - Every function returns 0 (CTAUX_OK) or a negative CTAUX_E* code; nothing aborts the process.
 *   - The caller owns every buffer it passes in.  `g0_table` and `seeds` are HOST pointers and are
 *     copied during the call.  `workspace` is a DEVICE pointer (e.g. a torch uint8 tensor) of at
 *     least ctaux_workspace_bytes() bytes, 256-byte aligned, which must stay alive and untouched
 *     until ctaux_destroy(); the context sub-allocates it and owns nothing else on the device.
 *   - `stream` is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); all kernels of
 *     the context are launched on it.  ctaux_sweep returns when the requested sweeps are done
 *     (it polls a completion flag, because the number of proposal blocks is data dependent);
 *     every ctaux_get_* synchronises the stream before reading.
 *   - Matrices handed out are column-major with the leading dimension the caller states, in the
 *     order of the walker's vertex LIST (ascending vertex id).
 *   - There is no CPU fallback: without a CUDA device every call returns CTAUX_ECUDA.
 */
#ifndef CTAUX_H_
#define CTAUX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CTAUX_OK 0
#define CTAUX_EINVAL (-1)     /* bad argument / inconsistent parameters                       */
#define CTAUX_ECAPACITY (-2)  /* a walker would exceed max_k, or the workspace is too small   */
#define CTAUX_ECUDA (-3)      /* CUDA runtime error (see ctaux_last_cuda_error)               */
#define CTAUX_ESINGULAR (-4)  /* A_sigma numerically singular during a rebuild                */
#define CTAUX_ESTATE (-5)     /* call not valid in this state (e.g. sweep before reset)       */

typedef struct ctaux_ctx ctaux_ctx; /* opaque */

/* Parameters of ctaux_create.  Names follow the paper's input file where one exists. */
typedef struct ctaux_params {
  int32_t Lx, Ly;          /* periodic cluster, Nc = Lx*Ly, site i = x + Lx*y      */
  double beta;             /* inverse temperature                                      */
  double U;                /* on-site Hubbard U >= 0; N_corr = Nc.  U = 0 (gamma = 0) is
                              accepted only where the fused small-k path runs (else CTAUX_EINVAL)      */
  double K;                /* CT-AUX expansion parameter K of Eq. (22)            */
  int32_t n_tau;           /* M = number of tau INTERVALS (`sp-time-intervals`);
                              the table has M+1 points per row                                        */
  const double* g0_table;  /* HOST, [Nc][M+1] row-major, STANDARD sign (G0 < 0 at r=0 on (0,beta)),
                              row d = displacement dx + Lx*dy, column m = tau_m = m*beta/M with
                              m=0 meaning 0+ and m=M meaning beta-                                    */
  int32_t delay;           /* max buffered ACCEPTED changes per block = rank of the flush
                              (`max-submatrix-size`).  Performance knob only:
                              the Markov chain does not depend on it.  1 <= delay <= 256             */
  int32_t n_walkers;       /* B independent chains batched on the device               */
  int32_t init_k;          /* random vertices drawn at reset (`initial-configuration-size`) */
  int32_t max_k;           /* capacity of the vertex list; exceeding it is CTAUX_ECAPACITY
                              (`initial-matrix-size` idea)                              */
  int32_t rebuild_every;   /* sweeps between from-scratch rebuilds of N (0 = never). Chain-neutral.   */
  int32_t log_capacity;    /* decision-log entries kept per walker (0 = logging off)                  */
  int32_t cand_window;     /* insertion candidates pre-expanded per block (0 = library default,
                              about 1.25*delay+8).  Performance knob only.                            */
  void* workspace;         /* DEVICE pointer, caller-owned                                            */
  size_t workspace_bytes;
  void* stream;            /* cudaStream_t                                                            */
  double guard_amp;        /* numerical guard of the delayed block: a block is
                              flushed BEFORE a proposal whose bordered ratio evaluation would amplify
                              rounding errors by more than guard_amp (cancellation in
                              s_nn - s_row S^-1 s_col, times the error level S^-1 already carries);
                              the proposal is then evaluated from the freshly updated N.  This
                              happens when A is nearly singular (e.g. while thermalising from the
                              random initial configuration).  0 = library default (100: ends ~1.5% of
                              the blocks early in equilibrium); < 0 or inf = off.  Chain-neutral: only where blocks
                              end.                                                                    */
  int32_t fused_small;     /* small-k path: 0 = automatic (used when both N_sigma of a walker fit one SM's
                              shared memory, max_k <= ~100), 1 = require it (CTAUX_ECAPACITY if it does not
                              fit), -1 = never.  The fused kernel runs whole sweeps of a walker in one launch
                              with N in shared memory and applies every accepted move at once (delay and
                              cand_window are ignored there: they are chain-neutral knobs).              */
  int32_t rebuild_mode;    /* periodic rebuild of N: 0 = from scratch, blocked LU with partial pivoting (the default and
                              what ctaux_reset / ctaux_set_state / ctaux_rebuild always do); 1 = refresh by one
                              Newton-Schulz step N <- N (2 - A N) with A rebuilt from the configuration -- two dense
                              FP64 GEMMs instead of the latency-bound LU; quadratic, so an N that has drifted to
                              1e-9 comes back to rounding level.  Falls back to LU when max|A N - 1| > 1e-4.
                              Chain-neutral like every rebuild.  Needs one more k x k buffer per matrix.     */
  int32_t flip_moves;      /* 1: auxiliary-spin FLIP as a third move (Fig. 5 (c)->(d)): move type =
                              (w6 * 3) >> 32 (0 insert, 1 remove, 2 flip), flip of the vertex at list position
                              (w1 * k) >> 32, R = prod_sigma det A'/det A.  0 (default): the two-move chain of
                              BASELINE.json.  This DOES change the chain (it is a different sampler).          */
  double n_tol;            /* accuracy the library HOLDS for every N_sigma it hands out, as a relative Frobenius error against
                              the exact inverse of A rebuilt from the configuration (BASELINE.json: 1e-10).  Fast updates of
                              an inverse amplify the error N already carries, at a data-dependent rate, so a fixed cadence
                              either wastes rebuilds or misses the bar: the library ESTIMATES the forward error of every
                              N_sigma on the device (a 4-probe Hutchinson estimate of |(N A - 1) N|_F / |N|_F: two passes
                              over N, A never stored) at the end of every ctaux_sweep call and every few block steps inside
                              it, and runs the from-scratch rebuild (S1 + S5) of the context when the estimate exceeds
                              n_tol / 3 at the end of a call (30 n_tol inside a call, where only the acceptance ratios depend
                              on it).  0 = library default 1e-10; < 0 = monitor off (fixed cadence `rebuild_every` only).
                              Chain-neutral like every rebuild.                                                            */
  int32_t n_pairs;         /* general density-density interaction between OPPOSITE spins (Eq. (19)-(21)
                              PAPER.md:174-182, model parameters U, V of PAPER.md:743-778):
                                H_int = sum_p U_p [ n_{a_p up} n_{b_p down} - (n_{a_p up} + n_{b_p down}) / 2 ]
                              over N_corr = n_pairs pairs p = (pair_a[p], pair_b[p], pair_U[p]): on-site repulsion a = b,
                              inter-site / inter-layer / inter-orbital V between opposite spins a != b.  A vertex is then
                              (p, tau, s): the `site` of configurations and logs is the PAIR index; cosh(gamma_p) =
                              1 + U_p beta N_corr / (2K) (Eq. (25)); N_up is built on the sites a_p, N_down on the sites
                              b_p, both stay k x k.  0 = the on-site Hubbard model (pair p = site p,
                              N_corr = Nc, coupling `U`).  Interactions between EQUAL spins (V': two rows of one N_sigma per
                              vertex) are not supported.                                                                    */
  const int32_t* pair_a;   /* HOST [n_pairs] site of the up electron of pair p (ignored when n_pairs = 0)                    */
  const int32_t* pair_b;   /* HOST [n_pairs] site of the down electron                                                       */
  const double* pair_U;    /* HOST [n_pairs] coupling U_p > 0                                                                */
  int32_t n_omega;         /* single-particle accumulator (S6): number N_w of positive
                              fermionic Matsubara frequencies w_n = (2n+1) pi / beta, n = 0..N_w-1 (`sp-fermionic-frequencies`).
                              0 = accumulator off (ctaux_accumulate returns CTAUX_ESTATE).                                  */
  int32_t nfft_oversampling;/* m of Eq. (31): the tau grid has m * N_w points.  0 = library default 4; >= 2. */
  int32_t nfft_window;     /* half-width w of the convolution kernel in grid cells (every sample touches 2w grid points,
                              2w <= 32).  0 = library default 6 (aliasing error ~2e-5 with m = 4; m = 8, w = 10: < 1e-9).   */
  int32_t graph_mode;      /* CUDA graph of one poll interval of block steps (8 block steps, ~100 launches, incl. the fork to
                              and join from the internal S3 stream), captured per context and grid size class and relaunched:
                              0 = library default (on where a block step is launch bound: max_k <= 512), 1 = on for every
                              size, -1 = off.  Never changes results; off while ctaux_timing_enable is on.                   */
} ctaux_params;

/* Per-walker counters.  flops are ALGORITHMIC (unpadded) counts of the GEMM steps. */
typedef struct ctaux_stats {
  uint64_t proposals;      /* proposal counter p of the chain (runs on across sweep calls)            */
  uint64_t next_id;        /* id the next accepted insertion will get                                 */
  int64_t acc_ins, acc_rem;/* accepted insertions / removals since reset                              */
  int64_t sweeps;          /* sweeps completed since reset                                            */
  int64_t blocks;          /* proposal blocks run                                                     */
  int64_t flushes;         /* blocks that ended in a rank-r flush (r > 0)                             */
  int64_t rebuilds;        /* from-scratch rebuilds                                                   */
  int64_t sum_rank;        /* sum of r over flushes                                                   */
  int32_t k;               /* current expansion order                                                 */
  int32_t sign;            /* sign of prod_sigma det A_sigma carried along the chain                  */
  double flops_cand;       /* S2: 2*m*k*k (rows) + 2*n*n*m (columns), both spins                      */
  double flops_flush;      /* S4: 2*k'*k'*r (the rank-r update itself), both spins                    */
  double flops_rebuild;    /* S5: 2*k^3 per spin                                                      */
  double min_margin;       /* min over proposals of |u - |R|| / |R|  (near-tie diagnostic, Q22)       */
  double sum_k;            /* sum over proposals of k before the proposal (for <k>)                   */
  double flops_usinv;      /* S4: 2*k'*r*r (U * S^-1), both spins                                     */
  int64_t guard_ends;      /* blocks ended early by the numerical guard (ctaux_params.guard_amp)      */
  int64_t acc_flip;        /* accepted auxiliary-spin flips since reset (flip_moves = 1)              */
  int64_t monitor_rebuilds;/* rebuilds triggered by the error monitor (ctaux_params.n_tol), included in `rebuilds` */
  double err_est;          /* last forward-error estimate of this walker's N (max over the two spins; 0 = none yet)  */
  double flops_cand_alg;   /* S2 as SURVEY 8d counts it: 2*m*k*k (rows) + 2*n*n*r_ins (columns of ACCEPTED inserts only)   */
} ctaux_stats;

/* One entry of the decision log (48 bytes). */
typedef struct ctaux_log_entry {
  uint64_t p;              /* proposal counter                                                        */
  int32_t type;            /* 0 insert, 1 remove, 2 flip                                              */
  int32_t arg;             /* insert: site; remove / flip: list position j (-1 when k == 0)           */
  double tau;              /* insert: proposed tau; remove: 0                                         */
  int32_t spin;            /* insert: proposed auxiliary spin; remove: 0                              */
  int32_t accepted;        /* 1 iff u < |R|                                                           */
  double R;                /* signed acceptance ratio: K/(k+1) or k/K times prod_sigma det A'/det A   */
  double u;                /* the uniform it was compared with                                        */
} ctaux_log_entry;

/* Device bytes ctaux_create needs for these parameters (workspace fields ignored). 0 on bad input. */
size_t ctaux_workspace_bytes(const ctaux_params* prm);

/* Build a context: copies the table to the device, precomputes e^{+-gamma} (Eq. (25)),
 * carves the workspace.  *out is NULL on failure. */
int ctaux_create(const ctaux_params* prm, ctaux_ctx** out);

/* (Re)start all walkers: walker w draws init_k vertices from Philox4x32-10 keyed by seeds[w]
 * (HOST array of n_walkers), builds A_sigma and N_sigma = A_sigma^{-1} (S1 + S5), sets the proposal
 * counter to 0. */
int ctaux_reset(ctaux_ctx* ctx, const uint64_t* seeds);

/* Start every walker from a given configuration instead (HOST arrays of n_walkers*max_k entries,
 * walker w at offset w*max_k, k[w] live entries; ids ascending).  Used to resume a chain. */
int ctaux_set_state(ctaux_ctx* ctx, const uint64_t* seeds, const int32_t* k, const uint64_t* id,
                    const int32_t* site, const double* tau, const int8_t* spin,
                    const uint64_t* next_id, const uint64_t* proposals);

/* Advance every walker by n_sweeps sweeps; a sweep is max(16, k at sweep start) proposals
 * (S2, S3, S4 per block; S5 every rebuild_every sweeps).  Continues each walker's stream. */
int ctaux_sweep(ctaux_ctx* ctx, int32_t n_sweeps);

/* Advance every walker by exactly n_proposals proposals (a partial sweep): the chain is a function of the proposal
 * counter only (Philox counter = p), so splitting it this way changes nothing but where blocks end.  For
 * callers that measure or check between sweeps; counted as one sweep in ctaux_stats.sweeps, does not advance the
 * rebuild cadence (rebuild_every counts ctaux_sweep sweeps); N is held to n_tol at return like after ctaux_sweep. */
int ctaux_propose(ctaux_ctx* ctx, int32_t n_proposals);

/* From-scratch rebuild of every walker's N from its configuration (S1 + S5), now. */
int ctaux_rebuild(ctaux_ctx* ctx);

/* Configuration of one walker in list order into HOST arrays with room for `cap` entries.
 * Any of id/site/tau/spin may be NULL. *k receives the expansion order. */
int ctaux_get_config(ctaux_ctx* ctx, int32_t walker, int32_t* k, uint64_t* id, int32_t* site,
                     double* tau, int8_t* spin, int32_t cap);

/* N_sigma of one walker (spin 0 = up, 1 = down): k x k, column-major, leading dimension ld >= k,
 * into a HOST buffer, rows/columns in list order.  This is the incrementally updated matrix. */
int ctaux_get_N(ctaux_ctx* ctx, int32_t walker, int32_t spin, double* N, int32_t ld);

/* Batched read-out (one synchronisation for the whole context).  k: HOST [n_walkers]; id / site / tau / spin:
 * HOST [n_walkers][max_k] (walker w at offset w*max_k, list order; entries at or beyond k[w] are unspecified), any of
 * them may be NULL.  One gather kernel, one copy per field, one synchronisation. */
int ctaux_get_config_all(ctaux_ctx* ctx, int32_t* k, uint64_t* id, int32_t* site, double* tau, int8_t* spin);

/* Every N_sigma of the context into one HOST buffer: matrix (w, spin) is k_w x k_w, column-major with leading
 * dimension k_w, at offset (2*w + spin) * max_k * max_k doubles.  `N` should be pinned for full PCIe rate. */
int ctaux_get_N_all(ctaux_ctx* ctx, double* N);

/* Same matrix, copied device-to-device into a DEVICE buffer (no host staging). */
int ctaux_get_N_device(ctaux_ctx* ctx, int32_t walker, int32_t spin, double* N_dev, int32_t ld);

int ctaux_get_stats(ctaux_ctx* ctx, int32_t walker, ctaux_stats* out);

/* Counters of every walker with one synchronisation and one copy: out is a HOST array of n_walkers ctaux_stats. */
int ctaux_get_stats_all(ctaux_ctx* ctx, ctaux_stats* out);

/* Copy log entries [first, first+count) of one walker into a HOST array; entries are numbered from
 * the last reset and the log keeps the first log_capacity of them. Returns the number copied (>=0). */
int64_t ctaux_get_log(ctaux_ctx* ctx, int32_t walker, ctaux_log_entry* out, int64_t first, int64_t count);

/* S6 -- single-particle accumulation, needs n_omega > 0.
 * ctaux_accumulate: for every walker and spin, M_sigma = (E - 1) N_sigma (factor on the row, so that
 * G_c = G0 - G0 M G0) of the CURRENT configuration, times the walker's sign, is convolved with the NFFT kernel onto the
 * context's tau grids (one per spin and displacement r_j - r_l; Eq. (30)-(31) PAPER.md:232-238) -- the delayed NFFT: no
 * transform happens here.  Asynchronous on the context stream.  Call it between ctaux_sweep calls
 * (`sweeps-per-measurement`).
 * ctaux_get_M: the ONE transform at the end: out[spin][r][n] = (1/phi_n) sum_l grid[spin][r][l] e^{i w_n l beta/L}
 * = sum over all accumulated configurations of sign * sum_{jl: r_j-r_l=r} M[j,l] e^{i w_n (tau_j - tau_l)}, as (re, im)
 * pairs into the HOST array M [2][Nc][n_omega][2]; *sign_sum = sum of the signs, *n_meas = configurations accumulated
 * (either may be NULL).  <M(r, iw_n)> = out / sign_sum; Eq. (28)-(29) then give G and Sigma.  Does not reset.
 * ctaux_reset_accumulator: zero the grids and counters. */
int ctaux_accumulate(ctaux_ctx* ctx);
int ctaux_get_M(ctaux_ctx* ctx, double* M, double* sign_sum, int64_t* n_meas);
int ctaux_reset_accumulator(ctaux_ctx* ctx);

/* Bare cluster propagator of the DCA: the table ctaux_create consumes, computed on the device from the
 * cluster self-energy instead of the isolated-cluster closed form.
 *   Gbar(K, iw_n) = patch average of [i w_n - eps_k + mu - Sigma_c(K, iw_n)]^-1   (Eq. (6)-(8) PAPER.md:85-93; standard
 *                   square patches of the periodic Lx x Ly cluster, n_quad x n_quad midpoint rule; n_quad = 1 = the
 *                   isolated cluster; eps_k = -2t (cos kx + cos ky), Eq. (45))
 *   G0c(K, iw_n)  = [Gbar^-1 + Sigma_c]^-1                                        (cluster exclusion, Eq. (9))
 *   table[d][m]   = G0c(r_d, m beta / n_tau), m = 0..n_tau (0+ and beta- at the ends), STANDARD sign, row d = dx + Lx dy:
 *                   (1/Nc) sum_K e^{iK.r}, Matsubara sum over +-n from the n_omega positive frequencies with the
 *                   three-moment tail summed analytically (truncation error O(n_omega^-3)).
 * sigma_c: HOST [Nc][n_omega][2] (re, im; K = 2 pi (nx/Lx, ny/Ly) at index nx + Lx ny; must obey Sigma_c(-K) = Sigma_c(K)),
 * or NULL for Sigma_c = 0.  table: HOST [Nc][n_tau + 1].  workspace: DEVICE scratch of ctaux_g0_workspace_bytes().
 * Synchronises the stream. */
size_t ctaux_g0_workspace_bytes(int32_t Lx, int32_t Ly, int32_t n_omega, int32_t n_tau);
int ctaux_g0_table(void* stream, int32_t Lx, int32_t Ly, double t, double mu, double beta, int32_t n_omega, int32_t n_quad,
                   const double* sigma_c, int32_t n_tau, double* table, void* workspace, size_t workspace_bytes);

/* ctaux_g0_table for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same operation (Eq. (6)-(9)), same kernels, same arguments and
 * results (sigma_c HOST or NULL, table HOST, synchronises the stream), but the scratch is a static device array inside
 * the library instead of a caller workspace; the call performs no cudaMalloc / cudaFree and calls no allocating library
 * routine.  Limits and sharing:
 *   - ctaux_g0_workspace_bytes(Lx, Ly, n_omega, n_tau) must not exceed CTAUX_G0_NOALLOC_MAX_BYTES (8 MiB: e.g. a 6x6
 *     cluster with n_omega = 2048, n_tau = 4096); larger sizes return CTAUX_ECAPACITY and ctaux_last_cuda_error() names
 *     the bytes needed.  Every GPU that loads the library holds the 8 MiB until the process exits.
 *   - ALL calls on a device share the one array: two calls that overlap on the GPU (different streams or host threads)
 *     race.  Serialise them.  The array keeps the last call's contents; every element a call reads is written earlier in
 *     that same call, so no clearing is needed and results do not depend on earlier calls.
 * Errors as ctaux_g0_table: CTAUX_EINVAL for invalid sizes / NULL table, CTAUX_ECUDA for CUDA failures. */
#define CTAUX_G0_NOALLOC_MAX_BYTES (8u << 20)
int ctaux_g0_table_noalloc(void* stream, int32_t Lx, int32_t Ly, double t, double mu, double beta, int32_t n_omega,
                           int32_t n_quad, const double* sigma_c, int32_t n_tau, double* table);

/* Kernel launches issued by this context since creation (bench.py's gpu_launches). */
int64_t ctaux_launch_count(ctaux_ctx* ctx);

/* Device time (ms, CUDA events on the context stream) spent in each step class since the last
 * ctaux_timing_reset: [0] S1+S2 prep, [1] S2 GEMMs, [2] S3 proposal, [3] S4 U/V build,
 * [4] S4 flush GEMMs, [5] S5 rebuild, [6] other.  Only filled when timing is enabled (it
 * serialises launches with events; off by default). */
int ctaux_timing_enable(ctaux_ctx* ctx, int32_t on);
int ctaux_timing_get(ctaux_ctx* ctx, double* ms /*[8]*/, int64_t* launches /*[8]*/);

void ctaux_destroy(ctaux_ctx* ctx);

const char* ctaux_strerror(int code);
const char* ctaux_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CTAUX_H_ */
