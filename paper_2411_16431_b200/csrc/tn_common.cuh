// Internal declarations shared by the translation units of libtn_b200.so.
// Product code: never includes or links anything under oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <cmath>
#include <string>
#include <vector>
#include <stdexcept>
#include "../../include/tn.h"

struct TnError {
  int code;
  std::string msg;
};
[[noreturn]] void tn_throw(int code, const char* fmt, ...);
#define TN_CUDA(expr)                                                                      \
  do {                                                                                     \
    cudaError_t e__ = (expr);                                                              \
    if (e__ != cudaSuccess)                                                                \
      tn_throw(e__ == cudaErrorMemoryAllocation ? TN_ERR_OOM : TN_ERR_CUDA, "%s: %s (%s:%d)", \
               #expr, cudaGetErrorString(e__), __FILE__, __LINE__);                        \
  } while (0)

typedef long long i64;

// ---------------------------------------------------------------------------------------------
// Per-cell tables (a1).  State spaces of a cell made of S sub-clusters A, B, C of n_s spins:
//   a in [0,nA)   sub-cluster 0 (carries the horizontal legs),
//   b in [0,nB)   the sub-cluster that carries the vertical legs (sub 1; for S == 1 it IS a),
//   c = c_lo + nCl*c_hi  sub-cluster 2 (S == 3): c_lo carries dout, c_hi carries din,
//   k = a*nCl + c_lo in [0,nK): the part of the state that indexes the horizontal MPO bonds.
// Cell weight  w(a,b,c) = g(k,b) * wC[c_lo][c_hi],   g(k,b) = wA[a] * X[a>>tshift][b] * Yc[b][c_lo].
// ---------------------------------------------------------------------------------------------
struct CellDev {
  int nA, nB, nT, nCl, nCh, nK, tshift;
  int n_l, n_r, n_u, n_d, n_i, n_o;   // projector ranges (Eq. (5))
  int bh_rows, bv_rows, bd_rows;      // rows of the incoming edge matrices (ranges of the neighbours)
  int m_left, m_right, m_din, m_dout; // coupled-bit masks (m_din relative to the hi half)
  int m_up, m_down;                   // coupled-bit masks of the vertical sub-cluster
  const double *wA, *X, *Yc, *wC;     // [nA] [nT*nB] [nB*nCl] [nCl*nCh]
  const int *Pl, *Pr, *Pu, *Pd, *Pi, *Po;  // [nA] [nA] [nB] [nB] [nCh] [nCl]
  const double *Bh, *Bv, *Bd;         // [bh_rows*n_l] [bv_rows*n_u] [bd_rows*n_i]
  const double *BhS, *BvS;            // [bh_rows*nA] [bv_rows*nB]  (columns expanded to states)
};

struct MpsTensor {
  double* d = nullptr;
  int dl = 1, p = 1, dr = 1;
};

struct Timer {
  cudaEvent_t a = nullptr, b = nullptr;
};

struct tn_handle {
  // instance
  int n_spins = 0;
  i64 n_edges = 0;
  int Ly = 0, Lx = 0, S = 0, ns = 0;
  std::vector<int> edge_u, edge_v, cell_of, bit_of;   // bit_of: sub*ns+pos
  std::vector<double> J, h;
  int *d_eu = nullptr, *d_ev = nullptr, *d_cell_of = nullptr, *d_bit_of = nullptr;
  double *d_J = nullptr, *d_h = nullptr;
  // table build inputs
  void* d_cell_edges = nullptr;
  int* d_cell_edge_ptr = nullptr;
  void* d_cell_desc = nullptr;
  // tables
  std::vector<CellDev> cells;   // host copy of the descriptors (pointers are device pointers)
  CellDev* d_cells = nullptr;
  double* pool_d = nullptr;
  int* pool_i = nullptr;
  double* d_offsets = nullptr;
  double beta = 0, offset = 0;
  bool have_beta = false, have_mps = false;
  // boundary MPS: rows[y] for y = 1..Ly (rows[Ly] trivial)
  std::vector<std::vector<MpsTensor>> rows;
  std::vector<double> lognorm;
  double log_z = 0;
  bool have_logz = false;
  int D = 0, sweeps = 0;
  // options
  int merge = 0;            // TN_OPT_MERGE: merge candidates by boundary before the bound (Fig. 3(d))
  double *lbp_nu = nullptr, *lbp_mu = nullptr;   // f4: LBP messages [cell][6][256] / [cell][7][256] (lbp.cu)
  bool have_lbp = false;
  int droplets = 0, droplet_min_hamming = 1, droplet_max_count = 8;   // TN_OPT_DROPLETS ... (Fig. 4)
  double droplet_max_dE = 1.0;
  std::vector<int> drop_cnt;          // results of the last tn_branch_and_bound: droplets per returned state,
  std::vector<double> drop_dE;        //   [state][K] excitation energies,
  std::vector<int8_t> drop_flips;     //   [state][K][n_spins] flip masks
  int drop_K = 0;
  int merge_segmented = 1;
  int ts_rpw3 = 1;          // TN_OPT_TS_WIDE_ROWS: 24-row warp tiles in k_tsgemm for 24..48 columns
  int lazy_v = 1;           // TN_OPT_LAZY_V: V is not written by k_cond; k_cond_rows writes the rows the selection reads
  int select_rows = 1;      // TN_OPT_SELECT_ROWS: selection bound and prefilter through the row maxima of V
  int rblock_fact = 1;      // TN_OPT_RBLOCK_FACT: factorised right-block contraction (k_rblock_h)
  int cond_pipe = 1;        // TN_OPT_COND_PIPE: pipelined conditional GEMM (k_cond) where the shape fits
  i64 merge_cap = 1ll << 20;  // TN_OPT_MERGE_CAP: survivors / boundary groups the merge buffers hold
  int gap_guard = 1, svd_maxit = 40, oversample = 16, exact_cap = 512, svd_cheb = 1, svd_lock = 1;
  int schedule = 0, sweep_range = 2, svd_mode = 0, rsvd_iters = 2, two_step = 0;   // f2 (TN_OPT_SCHEDULE ...)
  int svd_direct = 1;       // TN_OPT_SVD_DIRECT: explicit Theta + Jacobi SVD where Theta is tiny
  int svd_skip_first = 0;   // predictor (contract.cu): skip the first Rayleigh-Ritz step of the next truncated SVD
  double svd_tol = 1e-11;
  i64 select_direct_max = 1ll << 22;
  // runtime
  cudaStream_t stream = nullptr;
  void* (*alloc_cb)(size_t, void*) = nullptr;
  void (*free_cb)(void*, void*) = nullptr;
  void* alloc_ctx = nullptr;
  i64 bytes_held = 0;
  struct Block { void* p; size_t bytes; int src; unsigned long long serial; };   // src: 0 cudaMalloc, 1 allocator callback
  std::vector<Block> live, cached;
  unsigned long long serial = 0;   // allocation counter: every block handed out by dmalloc carries the value at its birth
  int device = 0, sms = 148;       // CUDA device of this handle and its SM count (queried at tn_create)
  tn_stats st;
  cudaEvent_t ev[2] = {nullptr, nullptr};
  unsigned long long* d_cnt = nullptr;   // device counters: [0] Jacobi calls, [1] Jacobi sweeps

  void* dmalloc(size_t bytes);
  void dfree(void* p);
  // error paths: every block handed out after `mark = serial` was taken goes back to the free list
  void release_since(unsigned long long mark);
  template <class T>
  T* dalloc(size_t n) { return (T*)dmalloc(n * sizeof(T) + 16); }
  const CellDev& cell(int y, int x) const { return cells[(size_t)y * Lx + x]; }
  bool has_med() const { return S == 3; }
};

// One-time (per device) opt-in to more than 48 KB of dynamic shared memory for kernel `fn`.
#define TN_SMEM_OPT_IN(h, fn, bytes)                                                                   \
  do {                                                                                                 \
    static bool done__[64] = {false};                                                                  \
    const int d__ = (h)->device & 63;                                                                  \
    if (!done__[d__]) {                                                                                \
      TN_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bytes)));    \
      done__[d__] = true;                                                                              \
    }                                                                                                  \
  } while (0)

// simple scoped device buffer
template <class T>
struct DBuf {
  tn_handle* h;
  T* p = nullptr;
  size_t n = 0;
  DBuf(tn_handle* h_, size_t n_) : h(h_), n(n_) { p = h->dalloc<T>(n_ ? n_ : 1); }
  ~DBuf() { if (p) h->dfree(p); }
  DBuf(const DBuf&) = delete;
  DBuf& operator=(const DBuf&) = delete;
  DBuf(DBuf&& o) : h(o.h), p(o.p), n(o.n) { o.p = nullptr; }
  T* release() { T* q = p; p = nullptr; return q; }
};

struct StageTimer {   // accumulates GPU milliseconds of a stage into a stats field (syncs at stop)
  tn_handle* h;
  double* dst;
  cudaEvent_t a, b;
  StageTimer(tn_handle* h_, double* dst_);
  ~StageTimer();
};

// ---- tables.cu
void tables_create(tn_handle* h);          // host preprocessing + device layout (tn_create)
void tables_set_beta(tn_handle* h, double beta);
void tables_destroy(tn_handle* h);
// ---- contract.cu
void contract_run(tn_handle* h, int D, int sweeps);
void mps_free(tn_handle* h);
// ---- search.cu
void search_logz(tn_handle* h);
void search_run(tn_handle* h, int M, int* n_out, int8_t* states, double* energies, double* logp,
                double* log_pd);
void energy_run(tn_handle* h, int n, const int8_t* states, double* energies);
// ---- tsgemm.cu: allocation-free Theta-core^T x skinny apply on device pointers (static device scratch)
void gemm_t_static_run(void* stream, i64 m, int n, i64 k, const double* A, i64 lda, const double* B, i64 ldb, double* C,
                       i64 ldc);
// ---- lbp.cu (f4: loopy belief propagation, Sec. IV)
void lbp_run(tn_handle* h, int iterations);
void lbp_free(tn_handle* h);
void lbp_message(tn_handle* h, int y, int x, int leg, int* n, double* out);
void lbp_marginals(tn_handle* h, int y, int x, i64 n, const unsigned* states, double* logp);
void lbp_select(tn_handle* h, int y, int x, int K, int* n_out, unsigned* states, double* logp);
// ---- orth.cu
void kernel_check_run(tn_handle* h, int op, i64 m, int n, int k, const double* A, const double* B, double* C);
void kernel_bench_run(tn_handle* h, int op, i64 m, int n, i64 k, int iters, double* ms_per_call);
