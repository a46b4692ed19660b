/* tn.h -- C ABI of the B200-native boundary-MPS / branch-and-bound hot path of
 * arXiv 2411.16431 (Dziubyna et al., "Limitations of tensor-network approaches for
 * optimization and sampling ...").  Citations are PAPER.md:<line> + section / equation.
 *
 * Problem (Eq. (1)):  H(s) = sum_<ij> J_ij s_i s_j + sum_i h_i s_i,  s_i = +-1,
 * on a quasi-2D graph whose spins are grouped into unit cells on an Ly x Lx grid (Eq. (3),
 * PAPER.md:69-74, Fig. 1).  The library samples low-energy states from the
 * Boltzmann distribution p ~ exp(-beta H) (Eq. (6)) by
 *   (1) tn_set_beta : local Boltzmann tables, projectors and edge matrices (Eqs. (3)-(5)
 *                     PAPER.md:69-84, Fig. 5(c)),
 *   (2) tn_contract : boundary-MPS contraction of the sparse PEPS, row after row, bond <= D
 *                     (zipper + truncated SVD + one-site variational passes,
 *                     Sec. III B 2 PAPER.md:165-179, Fig. 8; sparse diagrams Fig. 7
 *                     PAPER.md:155-163),
 *   (3) tn_branch_and_bound : beam search over cells driven by the conditional probabilities
 *                     of Fig. 6(b) PAPER.md:143 (Eqs. (7)-(9) PAPER.md:94-107, Fig. 3).
 *
 * Conventions
 *   - every entry point returns a tn_status (0 = TN_OK, < 0 = error); no exception, abort or
 *     exit crosses this boundary; tn_last_error() gives a thread-local message.
 *   - pointers marked HOST are host memory, read (inputs) or written (outputs) synchronously;
 *     inputs are copied at tn_create, the caller keeps ownership of everything it passes in;
 *     outputs are caller-allocated with the stated capacity.
 *   - a handle owns all its device memory; it is single-threaded; distinct handles are
 *     independent.  All work is queued on the stream given by tn_set_stream (default: the
 *     legacy default stream) and calls return after the stream has been synchronised
 *     (tn_contract / tn_branch_and_bound need host-side control flow anyway).
 *   - there is NO CPU fallback: without a CUDA device every compute call returns TN_ERR_CUDA.
 *   - call order: tn_create -> tn_set_beta -> tn_contract -> tn_log_z / tn_branch_and_bound;
 *     a call made too early returns TN_ERR_STATE.  tn_set_beta drops the boundary MPS.
 *
 * Geometry accepted by tn_create (BASELINE.json "Pegasus-/Zephyr-shaped" synthetic lattices):
 *   a cell is a chain of S = subs_per_cell (1..3) sub-clusters of n_s = spins_per_sub spins
 *   (2..8, even; with S == 1 any n_s in 1..8 -- n_s = 1 is the square lattice of App. B, one spin
 *   per site); lo = positions [0, n_s/2), hi = [n_s/2, n_s).  Allowed edges:
 *     inside a sub-cluster: any pair;   sub s hi -- sub s+1 lo  (same cell);
 *     horizontal (x,y)-(x+1,y): sub 0 -- sub 0;  vertical (x,y)-(x,y+1): sub v -- sub v with
 *     v = min(1, S-1);  diagonal (x,y)-(x+1,y+1) (S == 3 only): sub 2 lo -- sub 2 hi.
 *   Anything else (e.g. a real D-Wave working graph) returns TN_ERR_GEOMETRY.
 */
#ifndef TN_B200_H
#define TN_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tn_handle tn_handle; /* opaque */

typedef enum {
  TN_OK = 0,
  TN_ERR_ARG = -1,      /* NULL / out-of-range argument                         */
  TN_ERR_GEOMETRY = -2, /* edge or cluster map outside the accepted geometry     */
  TN_ERR_STATE = -3,    /* call order violated                                   */
  TN_ERR_CUDA = -4,     /* CUDA runtime error or no device                       */
  TN_ERR_OOM = -5,      /* device allocation failed                              */
  TN_ERR_NUMERIC = -6   /* NaN / Inf / non-convergence detected                  */
} tn_status;

/* option keys for tn_set_option */
enum {
  TN_OPT_GAP_GUARD = 1,   /* 1 (default) / 0: never cut between singular values closer than 1e-6
                             relative (reading S5)                                   */
  TN_OPT_SVD_TOL = 2,     /* residual tolerance of the truncated SVD relative to sigma_1
                             (default 1e-11; reading S1)            */
  TN_OPT_SVD_MAXIT = 3,   /* max block-subspace iterations per zipper step (default 40)       */
  TN_OPT_OVERSAMPLE = 4,  /* extra block columns of the subspace iteration (default 16)       */
  TN_OPT_EXACT_CAP = 5,   /* largest bond allowed when D <= 0 (default 512)                   */
  TN_OPT_SVD_CHEB = 7,    /* 1 (default) / 0: Chebyshev-filtered subspace steps inside the truncated SVD when the
                             block's Ritz values decay slowly (same converged subspace, fewer Theta applies)  */
  TN_OPT_SVD_LOCK = 8,    /* 1 (default) / 0: freeze converged leading Ritz triplets of the truncated SVD and apply
                             Theta only to the remaining columns (deflation; same converged subspace)          */
  TN_OPT_MERGE = 9,       /* 0 (default) / 1: merge candidates with the same boundary before the bound, keeping the
                             most probable one (Fig. 3(d); reading S11)                 */
  TN_OPT_MERGE_CAP = 10,  /* capacity of the merge buffers (survivors above the threshold resp. possible boundaries of a
                             cell; default 2^20, range 1..2^24).  A cell whose candidates fit neither route is selected
                             WITHOUT merging and counted in tn_stats.merge_fallback_cells                      */
  /* ---- f2: the paper's preferred contraction schedule (Sec. III B 2; readings S21-S23).
     The defaults (0) are the parity definition S1-S4: converged SVD, whole zipper first, then the passes. */
  TN_OPT_SCHEDULE = 11,   /* 0 (default): whole zipper, then `sweeps` passes (the paper's variant (ii));
                             1: every zipper step is followed by a variational sweep of the instantaneous stage of the
                             zipper over TN_OPT_SWEEP_RANGE positions right of the centre and back, then `sweeps`
                             global passes ("each step of the zipper procedure is followed by a sweep")  */
  TN_OPT_SWEEP_RANGE = 12,/* positions to the right of the zipper's centre inside the local sweep (default 2; "a few
                             tensors in the vicinity of the instantaneous centre")                              */
  TN_OPT_SVD_MODE = 13,   /* 0 (default): converged truncated SVD (reading S1); 1: truncated randomized SVD with a fixed
                             number of subspace iterations (refs [43, 44]): seeded, counter-based random
                             block, reproducible run to run -- fewer Theta applies, accuracy left to the passes   */
  TN_OPT_RSVD_ITERS = 14, /* subspace iterations of the randomized SVD (default 2)                             */
  TN_OPT_TWO_STEP = 15,   /* 0 (default) / 1: zipper and passes at bond 2 D, then canonical truncation to D
                             ("targeting 2 chi singular values ... further truncated to the target chi") */
  /* ---- f1: droplets = excitation bookkeeping on top of the merge (Fig. 4; reading S24) */
  TN_OPT_DROPLETS = 16,             /* 0 (default) / 1 (needs TN_OPT_MERGE): every main branch carries the low-energy
                                       excitations that merged into it; read them with tn_droplets               */
  TN_OPT_DROPLET_MAX_DE = 17,       /* energy cutoff of a droplet above its main branch (default 1.0)          */
  TN_OPT_DROPLET_MIN_HAMMING = 18,  /* minimal pairwise Hamming distance of the droplets kept on one branch (default 1) */
  TN_OPT_DROPLET_MAX_COUNT = 19,    /* droplets kept per branch (default 8, range 1..32)                        */
  TN_OPT_MERGE_SEGMENTED = 20,      /* 1 (default) / 0: allow the segmented arg-max route of the merge (taken when the possible
                                       boundaries of a cell fit TN_OPT_MERGE_CAP); 0 forces threshold + sort everywhere   */
  TN_OPT_SVD_DIRECT = 21,           /* 1 (default) / 0: where Theta is tiny (n <= 128, n m + n^2 <= 24000 entries) form it explicitly
                                       and take its SVD by one-sided Jacobi in one kernel instead of iterating            */
  TN_OPT_COND_PIPE = 22,            /* 1 (default) / 0: search conditionals through the pipelined kernel k_cond (0: the generic
                                       batched kernel, kept as the reference route for the kernel-level comparison)        */
  TN_OPT_TS_WIDE_ROWS = 23,         /* 1 (default) / 0: 24-row warp tiles in the streaming GEMM for 24..48 columns (tuning switch) */
  TN_OPT_RBLOCK_FACT = 24,          /* 1 (default) / 2 / 0: right blocks through the factorised contraction (sum over c_lo, then over b;
                                       1: on the FP64 tensor cores, 2: the plain-FMA kernel) instead of the joint GEMM over
                                       (b, c_lo) x (beam, a_hi) (0: reference route)                                            */
  TN_OPT_SELECT_ROWS = 25,          /* 1 (default) / 0: top-M bound from the row maxima of V written by the conditional kernel and a
                                       prefilter that reads only the rows that reach it (0: hashed 1/64 sample + full pass over V)  */
  TN_OPT_LAZY_V = 26,               /* 1 (default) / 0: the conditional kernel does not write V; once the selection bound is known
                                       the rows that reach it are recomputed and written (no merge / droplets; needs
                                       TN_OPT_SELECT_ROWS and the pipelined conditional kernel) */
  TN_OPT_SELECT_DIRECT_MAX = 6 /* top-M selection: candidate counts up to this run the radix passes straight on
                             all candidates; above it a hashed 1/64 sample gives a lower bound of the (M+1)-th
                             key first and one prefilter pass compacts the survivors (default 2^22)  */
};

/* Counters and timers filled by tn_get_stats (all since the last tn_set_beta). */
typedef struct {
  double ms_tables;          /* a1: local tables kernel                                     */
  double ms_contract;        /* a2-a4(i): whole tn_contract                                  */
  double ms_theta_build;     /*   Theta-core builds (gather + batched DxDxD + weights)       */
  double ms_theta_apply;     /*   Theta x skinny / Theta^T x skinny DMMA GEMMs               */
  double ms_orth_svd;        /*   orthonormalisation + Jacobi SVD                            */
  double ms_search;          /* a4(ii)-a5: whole tn_branch_and_bound                         */
  double ms_search_rblocks;  /*   right blocks at row starts                                 */
  double ms_search_cond;     /*   conditional-probability GEMM + scores                      */
  double ms_search_select;   /*   top-M radix selection                                      */
  double flop_theta_build;   /* algorithmic FLOP of the builds                              */
  double flop_theta_apply;   /* algorithmic FLOP of the skinny GEMMs                        */
  double bytes_theta_apply;  /* algorithmic bytes of the skinny GEMMs (one read of Theta)    */
  double flop_search;        /* algorithmic FLOP of the search GEMMs                        */
  double bytes_search_cond;  /* algorithmic bytes of the conditionals: one write of V (8 M n_b n_cl n_a per cell)  */
  double bytes_search_select;/* algorithmic bytes of the top-M selection: one read of V per prefilter pass + the 1/64 sample passes */
  double min_sigma_rel;      /* max over the truncated bonds of (smallest retained sigma / sigma_1):
                                the worst cut of Fig. 12(b); 0 if nothing was cut */
  int64_t svd_iterations;    /* total block-subspace iterations                             */
  int64_t kernel_launches;   /* kernels launched by this library                            */
  int64_t negative_u;        /* conditionals clamped to 0 (reading S7)         */
  int64_t rows_contracted;   /* boundary-MPS rows built                                      */
  int64_t bytes_device;      /* device bytes currently held                                  */
  int64_t jacobi_calls;      /* one-sided Jacobi kernel launches                             */
  int64_t jacobi_sweeps;     /* total Jacobi sweeps over all calls                           */
  int64_t theta_apply_calls; /* Theta-core x skinny GEMM calls (launches of the dominant kernel)  */
  int64_t cheb_steps;        /* total Chebyshev degrees spent in filtered subspace steps           */
  int64_t svd_locked_cols;   /* Ritz triplets frozen by the locked subspace iteration (summed over all SVDs)        */
  int64_t merged_away;       /* candidates removed by TN_OPT_MERGE among those above the selection threshold        */
  int64_t svd_unconverged;   /* truncated SVDs stopped by TN_OPT_SVD_MAXIT with a residual above tolerance:
                                parity with a converged SVD (reading S1) is not guaranteed at those bonds  */
  int64_t merge_fallback_cells; /* cells at which TN_OPT_MERGE could not merge (merge buffers too small at every threshold
                                tried) and the selection ran unmerged; 0 = every cell followed Fig. 3(d)          */
  int64_t select_tie_overflow; /* cells whose tie group at the beam cut exceeded the candidate list and was collected completely */
  int64_t select_tie_dropped;  /* cells whose tie group exceeded even 2^24 candidates: an arbitrary subset of it was kept     */
  int64_t svd_direct;        /* truncated SVDs taken by the direct route (TN_OPT_SVD_DIRECT)                              */
  int64_t droplet_overflow;  /* boundary groups whose droplet candidates exceeded the kernel's buffer (1024): 0 = none     */
  double flop_orth_svd;      /* algorithmic FLOP of the orthonormalisations: 2 Cholesky-QR rounds of 4 m k^2 each per call
                                (Gram + apply; the rounds actually run are decided on the device, 1..5)             */
  double flop_search_rblocks;/* algorithmic FLOP of the right-block GEMMs (part of flop_search)                      */
  double flop_search_cond;   /* algorithmic FLOP of the conditional GEMMs LG and V (part of flop_search)             */
} tn_stats;

/* tn_create: validates the geometry and copies the instance to the device.
 *   n_spins, n_edges; edge_u/edge_v/J HOST [n_edges] (Eq. (1)); h HOST [n_spins] or NULL (= 0);
 *   Ly, Lx: cell grid (y = row, 0 = top; x = column, 0 = left);
 *   cell_y/cell_x/sub/pos HOST [n_spins]: cluster map (cell, sub-cluster in the cell, bit position
 *   in the sub-cluster; each (cell, sub, pos) slot holds exactly one spin; Eq. (3)).
 * Errors: TN_ERR_ARG, TN_ERR_GEOMETRY (message names the offending edge), TN_ERR_CUDA, TN_ERR_OOM. */
int tn_create(tn_handle** out, int32_t n_spins, int64_t n_edges,
              const int32_t* edge_u, const int32_t* edge_v, const double* J, const double* h,
              int32_t Ly, int32_t Lx, int32_t subs_per_cell, int32_t spins_per_sub,
              const int32_t* cell_y, const int32_t* cell_x, const int32_t* sub, const int32_t* pos);

/* tn_set_stream: cudaStream_t to launch on (borrowed; NULL = default stream). */
int tn_set_stream(tn_handle*, void* cuda_stream);

/* tn_set_allocator: device allocator callbacks (e.g. torch's caching allocator); must be set
 * before tn_set_beta; alloc returns NULL on failure; NULL callbacks restore cudaMalloc/cudaFree
 * (TN_ERR_STATE if blocks obtained from the previous callbacks are still live). */
int tn_set_allocator(tn_handle*, void* (*alloc)(size_t bytes, void* ctx),
                     void (*free_)(void* ptr, void* ctx), void* ctx);

int tn_set_option(tn_handle*, int32_t key, double value);

/* tn_set_beta (a1): Boltzmann weights exp(-beta (E - min E)) of every sub-cluster and
 * inter-sub-cluster table, projector index tables (Eq. (5)), edge matrices
 * exp(-beta (Ebar - min)) (Eq. (4), Fig. 5(c)).  Drops boundary MPS. */
int tn_set_beta(tn_handle*, double beta);

/* tn_contract (a2-a4): boundary MPS R_y for y = Ly-1 .. 1 with bond <= D, `sweeps` one-site
 * variational passes after each zipper.  D <= 0: no truncation (exact;
 * TN_ERR_ARG if a bond would exceed TN_OPT_EXACT_CAP), sweeps ignored. */
int tn_contract(tn_handle*, int32_t D, int32_t sweeps);

/* tn_log_z: log Z (Eq. (10)) from the contraction + the first cell's normaliser. */
int tn_log_z(tn_handle*, double* log_z /* HOST */);

/* tn_row_lognorm: log of the norm removed from R_y (y in 1..Ly-1), for row-wise parity. */
int tn_row_lognorm(tn_handle*, int32_t y, double* lognorm /* HOST */);

/* tn_mps_shape / tn_mps_tensor: copy boundary-MPS tensor `j` of R_y to the host, layout
 * [left bond][physical][right bond] row-major (padding directions are exactly zero). */
int tn_mps_shape(tn_handle*, int32_t y, int32_t j, int32_t* n_pos, int32_t* dl, int32_t* p, int32_t* dr);
int tn_mps_tensor(tn_handle*, int32_t y, int32_t j, double* out /* HOST dl*p*dr */);

/* tn_branch_and_bound (a4(ii)-a5): beam of width M over cells in row-major order (Fig. 3
 * PAPER.md:125).  Outputs (HOST, caller-allocated): *n_out <= M states; states [M][n_spins] int8
 * +-1 in spin-id order; energies [M] recomputed from J, h in input order (one running fp64
 * sum: edges first, then fields); logp [M] descending; *log_p_discarded = log of the largest
 * discarded probability p_d (-inf if nothing was discarded; may be NULL).
 * Ties: logp desc, then parent rank asc, then cell state asc (reading S8). */
int tn_branch_and_bound(tn_handle*, int32_t M, int32_t* n_out, int8_t* states, double* energies,
                        double* logp, double* log_p_discarded);

/* tn_droplets (f1, Fig. 4): the excitations book-kept above returned state `rank` of the last
 * tn_branch_and_bound (needs TN_OPT_MERGE and TN_OPT_DROPLETS; TN_ERR_STATE otherwise).  *n <= TN_OPT_DROPLET_MAX_COUNT;
 * dE HOST [max_count]: energy of main (+) flip above main, from the ratio of the marginals (increasing); flips HOST
 * [max_count][n_spins] int8: 1 = the droplet flips that spin.  Either output may be NULL. */
int tn_droplets(tn_handle*, int32_t rank, int32_t* n, double* dE, int8_t* flips);

int tn_get_stats(tn_handle*, tn_stats* out /* HOST */);

/* tn_energy: O-0 fixed-order energies of n given states (HOST int8 [n][n_spins]) on the device. */
int tn_energy(tn_handle*, int32_t n, const int8_t* states, double* energies /* HOST [n] */);

/* tn_kernel_check: diagnostic -- runs ONE device building block of the path on host data (kernel-level parity
 * tests call it; it is not a step of the path).  A, B, C are HOST row-major fp64.
 *   op = TN_CHECK_ORTH   : C [m x k] = orthonormalised columns of A [m x k] (a3: QR canonicalisation; n, B unused)
 *   op = TN_CHECK_GEMM_N : C [m x n] = A [m x k] . B [k x n]    (a2: Theta-core x skinny apply)
 *   op = TN_CHECK_GEMM_T : C [k x n] = A^T . B,  A [m x k], B [m x n]   (a2: Theta-core^T x skinny apply) */
enum { TN_CHECK_ORTH = 1, TN_CHECK_GEMM_N = 2, TN_CHECK_GEMM_T = 3 };
int tn_kernel_check(tn_handle*, int32_t op, int64_t m, int32_t n, int32_t k, const double* A, const double* B,
                    double* C);

/* tn_kernel_bench: diagnostic -- device time (CUDA events on the handle's stream, one untimed warm-up call) of one
 * building block on device-resident random data, averaged over `iters` calls, in ms per call:
 *   TN_CHECK_GEMM_N / TN_CHECK_GEMM_T with the shapes of tn_kernel_check (2 m n k FLOP per call, one read of A);
 *   TN_CHECK_ORTH: orthonormalisation of a random [m x n] block (k unused). */
int tn_kernel_bench(tn_handle*, int32_t op, int64_t m, int32_t n, int64_t k, int32_t iters, double* ms_per_call);

/* ---- f4: local dimensional reduction by loopy belief propagation (Sec. IV, Eqs. (11)-(13), Fig. 9).
 * tn_lbp: `iterations` rounds of [all cluster -> edge messages, Eq. (11); all edge -> cluster messages, Eq. (12)] from
 *   uniform messages, then the normalisers of Eq. (13); needs tn_set_beta; results stay on the
 *   handle until the next tn_set_beta (reading S26).
 * tn_lbp_message: the message arriving at cell (y, x) over leg 0 left, 1 right, 2 up, 3 down, 4 din, 5 dout: *n values
 *   (<= 256, the range of the leg's projector), normalised to sum 1 (constant 1 where there is no neighbour).
 * tn_lbp_marginals: log of the normalised LBP marginal p(x_n), Eq. (13), at n given states of cell (y, x)
 *   (HOST uint32: bit sub*n_s + pos = that spin, as in the cluster map).
 * tn_lbp_select: the K most probable states of cell (y, x) according to LBP ("we select the desired number
 *   of most probable states in each cluster"): *n_out = min(K, d) states, p descending, ties by ascending state.
 * The selection is reported; the contraction of this library keeps the full (factorised) cells. */
int tn_lbp(tn_handle*, int32_t iterations);
int tn_lbp_message(tn_handle*, int32_t y, int32_t x, int32_t leg, int32_t* n, double* nu /* HOST [256] */);
int tn_lbp_marginals(tn_handle*, int32_t y, int32_t x, int64_t n, const uint32_t* cell_states /* HOST [n] */,
                     double* logp /* HOST [n] */);
int tn_lbp_select(tn_handle*, int32_t y, int32_t x, int32_t K, int32_t* n_out, uint32_t* cell_states /* HOST [K] */,
                  double* logp /* HOST [K] */);

/* tn_gemm_t_static: ALLOCATION-FREE variant of the Theta-core^T x skinny apply (a2, Fig. 7), for callers
 * that cannot call cudaMalloc (CUDA graph capture, tight serving loops):  C [k x n] = A [m x k]^T . B [m x n],  all three
 * DEVICE pointers, row-major with leading dimensions lda >= k, ldb >= n, ldc >= n (lda, ldb even; A, B 16-byte aligned),
 * n <= 96.  Needs no handle.  The split-over-m workspace lives in a file-scope device array of 2^20 doubles (8 MiB, held by
 * every GPU that loads the library): sizes with 2 k n > 2^20 return TN_ERR_ARG.  The call queues two kernels on
 * `cuda_stream` (NULL = default stream) and returns without synchronising; it calls no cudaMalloc / cudaFree.  Every call
 * shares the scratch array: calls that overlap on the GPU (other streams, parallel graph branches) race on it. */
int tn_gemm_t_static(void* cuda_stream, int64_t m, int32_t n, int64_t k, const double* dA, int64_t lda, const double* dB,
                     int64_t ldb, double* dC, int64_t ldc);

/* tn_fp64_peak: measured FP64 tensor-core (mma.sync m8n8k4 f64 = SASS DMMA) peak of the current device
 * in TFLOP/s, from a register-resident chain (about 10 ms); the roofline denominator of the GEMM stages
 * ("FP64 tensor peak to be measured first").  Needs no handle. */
int tn_fp64_peak(double* tflops /* HOST */);

const char* tn_last_error(void);
void tn_destroy(tn_handle*);

#ifdef __cplusplus
}
#endif
#endif /* TN_B200_H */
