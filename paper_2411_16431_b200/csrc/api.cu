// C ABI of libtn_b200.so (include/tn.h).  No exception crosses this file's extern "C" functions.
#include "kernels.cuh"
#include <cstdarg>
#include <algorithm>

static thread_local std::string g_last_error;

[[noreturn]] void tn_throw(int code, const char* fmt, ...) {
  char buf[1024];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  throw TnError{code, buf};
}

// ---- device memory: allocator callbacks + a size-bucketed free list (all use is stream-ordered) ----
static void* raw_alloc(tn_handle* h, size_t bytes, int* src) {
  void* p = nullptr;
  if (h->alloc_cb) {
    p = h->alloc_cb(bytes, h->alloc_ctx);
    if (!p) tn_throw(TN_ERR_OOM, "allocator callback failed for %zu bytes", bytes);
    *src = 1;
  } else {
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) {
      cudaGetLastError();
      tn_throw(e == cudaErrorMemoryAllocation ? TN_ERR_OOM : TN_ERR_CUDA, "cudaMalloc(%zu): %s", bytes,
               cudaGetErrorString(e));
    }
    *src = 0;
  }
  return p;
}
static void raw_free(tn_handle* h, const tn_handle::Block& b) {
  if (b.src == 1 && h->free_cb) h->free_cb(b.p, h->alloc_ctx);
  else if (b.src == 0) cudaFree(b.p);
}
static void trim_free_list(tn_handle* h) {
  if (h->cached.empty()) return;
  cudaStreamSynchronize(h->stream);
  for (auto& b : h->cached) { raw_free(h, b); h->bytes_held -= (i64)b.bytes; }
  h->cached.clear();
}

void* tn_handle::dmalloc(size_t bytes) {
  bytes = (bytes + 255) & ~(size_t)255;
  auto& fl = cached;
  int best = -1;
  for (int i = 0; i < (int)fl.size(); i++)
    if (fl[i].bytes >= bytes && fl[i].bytes <= 2 * bytes + 4096 && (best < 0 || fl[i].bytes < fl[best].bytes)) best = i;
  Block blk;
  if (best >= 0) {
    blk = fl[best];
    fl.erase(fl.begin() + best);
  } else {
    try {
      blk.p = raw_alloc(this, bytes, &blk.src);
    } catch (TnError&) {
      trim_free_list(this);
      blk.p = raw_alloc(this, bytes, &blk.src);
    }
    blk.bytes = bytes;
    bytes_held += (i64)bytes;
  }
  blk.serial = ++serial;
  live.push_back(blk);
  return blk.p;
}
void tn_handle::dfree(void* p) {
  if (!p) return;
  for (size_t i = live.size(); i-- > 0;)
    if (live[i].p == p) {
      cached.push_back(live[i]);
      live[i] = live.back();
      live.pop_back();
      return;
    }
}

void tn_handle::release_since(unsigned long long mark) {
  for (size_t i = live.size(); i-- > 0;)
    if (live[i].serial > mark) {
      cached.push_back(live[i]);
      live[i] = live.back();
      live.pop_back();
    }
}

StageTimer::StageTimer(tn_handle* h_, double* dst_) : h(h_), dst(dst_) {
  cudaEventCreate(&a); cudaEventCreate(&b);
  cudaEventRecord(a, h->stream);
}
StageTimer::~StageTimer() {
  cudaEventRecord(b, h->stream);
  cudaEventSynchronize(b);
  float ms = 0;
  if (cudaEventElapsedTime(&ms, a, b) == cudaSuccess) *dst += ms;
  cudaEventDestroy(a); cudaEventDestroy(b);
}

#define TN_API_BEGIN try {
#define TN_API_END                                                     \
  return TN_OK;                                                        \
  }                                                                    \
  catch (const TnError& e) { g_last_error = e.msg; return e.code; }    \
  catch (const std::bad_alloc&) { g_last_error = "host out of memory"; return TN_ERR_OOM; } \
  catch (const std::exception& e) { g_last_error = e.what(); return TN_ERR_ARG; }            \
  catch (...) { g_last_error = "unknown error"; return TN_ERR_ARG; }

// Every entry point that touches the device runs on the handle's own device (a process may hold handles on several).
struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(const tn_handle* h) {
    if (h && cudaGetDevice(&prev) == cudaSuccess && prev != h->device) cudaSetDevice(h->device);
    else prev = -1;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

static void need_device() {
  int n = 0;
  cudaError_t e = cudaGetDeviceCount(&n);
  if (e != cudaSuccess || n == 0) {
    cudaGetLastError();
    tn_throw(TN_ERR_CUDA, "no CUDA device (%s); this library has no CPU fallback", cudaGetErrorString(e));
  }
}

extern "C" {

const char* tn_last_error(void) { return g_last_error.c_str(); }

int tn_create(tn_handle** out, int32_t n_spins, int64_t n_edges, const int32_t* edge_u, const int32_t* edge_v,
              const double* J, const double* hfield, int32_t Ly, int32_t Lx, int32_t S, int32_t ns,
              const int32_t* cell_y, const int32_t* cell_x, const int32_t* sub, const int32_t* pos) {
  tn_handle* h = nullptr;
  try {
    if (!out) tn_throw(TN_ERR_ARG, "out is NULL");
    *out = nullptr;
    if (n_spins <= 0 || n_edges < 0 || Ly <= 0 || Lx <= 0) tn_throw(TN_ERR_ARG, "non-positive size");
    if ((n_edges > 0 && (!edge_u || !edge_v || !J)) || !cell_y || !cell_x || !sub || !pos)
      tn_throw(TN_ERR_ARG, "NULL input array");
    if (S < 1 || S > 3 || ns < 1 || ns > 8 || (S > 1 && (ns & 1)))
      tn_throw(TN_ERR_GEOMETRY, "subs_per_cell must be 1..3 and spins_per_sub in 1..8, even unless subs_per_cell == 1 "
               "(got %d, %d)", S, ns);
    if ((i64)n_spins != (i64)Ly * Lx * S * ns)
      tn_throw(TN_ERR_GEOMETRY, "n_spins = %d but the cluster map has Ly*Lx*S*n_s = %lld slots", n_spins,
               (long long)Ly * Lx * S * ns);
    need_device();
    h = new tn_handle();
    memset(&h->st, 0, sizeof(h->st));
    h->n_spins = n_spins; h->n_edges = n_edges; h->Ly = Ly; h->Lx = Lx; h->S = S; h->ns = ns;
    h->edge_u.assign(edge_u, edge_u + n_edges);
    h->edge_v.assign(edge_v, edge_v + n_edges);
    h->J.assign(J, J + n_edges);
    h->h.assign(n_spins, 0.0);
    if (hfield) h->h.assign(hfield, hfield + n_spins);
    h->cell_of.resize(n_spins); h->bit_of.resize(n_spins);
    std::vector<char> used((size_t)n_spins, 0);
    for (int i = 0; i < n_spins; i++) {
      if (cell_y[i] < 0 || cell_y[i] >= Ly || cell_x[i] < 0 || cell_x[i] >= Lx || sub[i] < 0 || sub[i] >= S ||
          pos[i] < 0 || pos[i] >= ns)
        tn_throw(TN_ERR_GEOMETRY, "spin %d: cluster map entry out of range", i);
      h->cell_of[i] = cell_y[i] * Lx + cell_x[i];
      h->bit_of[i] = sub[i] * ns + pos[i];
      size_t slot = (size_t)h->cell_of[i] * S * ns + h->bit_of[i];
      if (used[slot]) tn_throw(TN_ERR_GEOMETRY, "spin %d: (cell, sub, pos) slot already taken", i);
      used[slot] = 1;
    }
    for (i64 e = 0; e < n_edges; e++) {
      if (edge_u[e] < 0 || edge_u[e] >= n_spins || edge_v[e] < 0 || edge_v[e] >= n_spins)
        tn_throw(TN_ERR_ARG, "edge %lld: spin index out of range", (long long)e);
      if (!std::isfinite(J[e])) tn_throw(TN_ERR_ARG, "edge %lld: J is not finite", (long long)e);
    }
    if (hfield)
      for (int i = 0; i < n_spins; i++)
        if (!std::isfinite(hfield[i])) tn_throw(TN_ERR_ARG, "spin %d: h is not finite", i);
    TN_CUDA(cudaGetDevice(&h->device));
    TN_CUDA(cudaDeviceGetAttribute(&h->sms, cudaDevAttrMultiProcessorCount, h->device));
    tables_create(h);
    h->d_eu = h->dalloc<int>(n_edges + 1); h->d_ev = h->dalloc<int>(n_edges + 1);
    h->d_J = h->dalloc<double>(n_edges + 1); h->d_h = h->dalloc<double>(n_spins);
    h->d_cell_of = h->dalloc<int>(n_spins); h->d_bit_of = h->dalloc<int>(n_spins);
    if (n_edges) {
      TN_CUDA(cudaMemcpy(h->d_eu, h->edge_u.data(), sizeof(int) * n_edges, cudaMemcpyHostToDevice));
      TN_CUDA(cudaMemcpy(h->d_ev, h->edge_v.data(), sizeof(int) * n_edges, cudaMemcpyHostToDevice));
      TN_CUDA(cudaMemcpy(h->d_J, h->J.data(), sizeof(double) * n_edges, cudaMemcpyHostToDevice));
    }
    TN_CUDA(cudaMemcpy(h->d_h, h->h.data(), sizeof(double) * n_spins, cudaMemcpyHostToDevice));
    TN_CUDA(cudaMemcpy(h->d_cell_of, h->cell_of.data(), sizeof(int) * n_spins, cudaMemcpyHostToDevice));
    TN_CUDA(cudaMemcpy(h->d_bit_of, h->bit_of.data(), sizeof(int) * n_spins, cudaMemcpyHostToDevice));
    h->d_cnt = h->dalloc<unsigned long long>(2);
    TN_CUDA(cudaMemset(h->d_cnt, 0, 2 * sizeof(unsigned long long)));
    *out = h;
    return TN_OK;
  } catch (const TnError& e) {
    g_last_error = e.msg;
    if (h) tn_destroy(h);
    return e.code;
  } catch (const std::exception& e) {
    g_last_error = e.what();
    if (h) tn_destroy(h);
    return TN_ERR_ARG;
  }
}

int tn_set_stream(tn_handle* h, void* s) {
  TN_API_BEGIN
  if (!h) tn_throw(TN_ERR_ARG, "handle is NULL");
  h->stream = (cudaStream_t)s;
  TN_API_END
}

int tn_set_allocator(tn_handle* h, void* (*alloc)(size_t, void*), void (*free_)(void*, void*), void* ctx) {
  TN_API_BEGIN
  if (!h) tn_throw(TN_ERR_ARG, "handle is NULL");
  if ((alloc == nullptr) != (free_ == nullptr)) tn_throw(TN_ERR_ARG, "alloc and free must both be set or both NULL");
  if (h->have_beta) tn_throw(TN_ERR_STATE, "tn_set_allocator must precede tn_set_beta");
  DeviceGuard dg(h);
  trim_free_list(h);   // blocks already handed out keep the origin they were allocated with (NULL, NULL = cudaMalloc again)
  if (h->alloc_cb != alloc || h->alloc_ctx != ctx)
    for (auto& l : h->live)
      if (l.src == 1) tn_throw(TN_ERR_STATE, "blocks from the previous allocator callbacks are still live");
  h->alloc_cb = alloc; h->free_cb = free_; h->alloc_ctx = ctx;
  TN_API_END
}

int tn_set_option(tn_handle* h, int32_t key, double v) {
  TN_API_BEGIN
  if (!h) tn_throw(TN_ERR_ARG, "handle is NULL");
  switch (key) {
    case TN_OPT_GAP_GUARD: h->gap_guard = v != 0.0; break;
    case TN_OPT_SVD_TOL:
      if (!(v > 0.0)) tn_throw(TN_ERR_ARG, "svd tol must be > 0");
      h->svd_tol = v; break;
    case TN_OPT_SVD_MAXIT:
      if (v < 1) tn_throw(TN_ERR_ARG, "maxit must be >= 1");
      h->svd_maxit = (int)v; break;
    case TN_OPT_OVERSAMPLE:
      if (v < 0 || v > 256) tn_throw(TN_ERR_ARG, "oversample out of range");
      h->oversample = (int)v; break;
    case TN_OPT_EXACT_CAP:
      if (v < 1 || v > 1024) tn_throw(TN_ERR_ARG, "exact cap must be in 1..1024");
      h->exact_cap = (int)v; break;
    case TN_OPT_SVD_CHEB: h->svd_cheb = v != 0.0; break;
    case TN_OPT_SVD_LOCK: h->svd_lock = v != 0.0; break;
    case TN_OPT_MERGE: h->merge = v != 0.0; break;
    case TN_OPT_SCHEDULE:
      if (v != 0.0 && v != 1.0) tn_throw(TN_ERR_ARG, "schedule must be 0 or 1");
      h->schedule = (int)v; break;
    case TN_OPT_SWEEP_RANGE:
      if (v < 0 || v > 1e6) tn_throw(TN_ERR_ARG, "sweep range must be >= 0");
      h->sweep_range = (int)v; break;
    case TN_OPT_SVD_MODE:
      if (v != 0.0 && v != 1.0) tn_throw(TN_ERR_ARG, "svd mode must be 0 or 1");
      h->svd_mode = (int)v; break;
    case TN_OPT_RSVD_ITERS:
      if (v < 1 || v > 100) tn_throw(TN_ERR_ARG, "randomized SVD iterations must be in 1..100");
      h->rsvd_iters = (int)v; break;
    case TN_OPT_TWO_STEP: h->two_step = v != 0.0; break;
    case TN_OPT_DROPLETS: h->droplets = v != 0.0; break;
    case TN_OPT_DROPLET_MAX_DE:
      if (!(v >= 0.0) || !std::isfinite(v)) tn_throw(TN_ERR_ARG, "droplet energy cutoff must be finite and >= 0");
      h->droplet_max_dE = v; break;
    case TN_OPT_DROPLET_MIN_HAMMING:
      if (v < 0 || v > 1e6) tn_throw(TN_ERR_ARG, "droplet Hamming threshold out of range");
      h->droplet_min_hamming = (int)v; break;
    case TN_OPT_DROPLET_MAX_COUNT:
      if (v < 1 || v > 32) tn_throw(TN_ERR_ARG, "droplets per branch must be in 1..32");
      h->droplet_max_count = (int)v; break;
    case TN_OPT_TS_WIDE_ROWS: h->ts_rpw3 = v != 0.0; break;
    case TN_OPT_SELECT_ROWS: h->select_rows = v != 0.0; break;
    case TN_OPT_LAZY_V: h->lazy_v = v != 0.0; break;
    case TN_OPT_RBLOCK_FACT: h->rblock_fact = v == 2.0 ? 2 : v != 0.0; break;
    case TN_OPT_COND_PIPE: h->cond_pipe = v != 0.0; break;
    case TN_OPT_SVD_DIRECT: h->svd_direct = v != 0.0; break;
    case TN_OPT_MERGE_SEGMENTED: h->merge_segmented = v != 0.0; break;
    case TN_OPT_MERGE_CAP:
      if (v < 1 || v > (double)(1 << 24)) tn_throw(TN_ERR_ARG, "merge cap must be in 1..2^24");
      h->merge_cap = (i64)v; break;
    case TN_OPT_SELECT_DIRECT_MAX:
      if (v < 0) tn_throw(TN_ERR_ARG, "select direct max must be >= 0");
      h->select_direct_max = (i64)v; break;
    default: tn_throw(TN_ERR_ARG, "unknown option key %d", key);
  }
  TN_API_END
}

int tn_set_beta(tn_handle* h, double beta) {
  TN_API_BEGIN
  if (!h) tn_throw(TN_ERR_ARG, "handle is NULL");
  if (!std::isfinite(beta) || beta < 0.0) tn_throw(TN_ERR_ARG, "beta must be finite and >= 0");
  DeviceGuard dg(h);
  mps_free(h);
  h->have_lbp = false;
  memset(&h->st, 0, sizeof(h->st));
  if (h->d_cnt) TN_CUDA(cudaMemsetAsync(h->d_cnt, 0, 2 * sizeof(unsigned long long), h->stream));
  tables_set_beta(h, beta);
  h->have_beta = true;
  TN_API_END
}

int tn_contract(tn_handle* h, int32_t D, int32_t sweeps) {
  TN_API_BEGIN
  if (!h) tn_throw(TN_ERR_ARG, "handle is NULL");
  if (!h->have_beta) tn_throw(TN_ERR_STATE, "tn_contract before tn_set_beta");
  if (sweeps < 0) tn_throw(TN_ERR_ARG, "sweeps < 0");
  if (D > 1008 || (h->two_step && D > 504)) tn_throw(TN_ERR_ARG, "D > 1008 (504 with TN_OPT_TWO_STEP) not supported");
  DeviceGuard dg(h);
  const unsigned long long mark = h->serial;
  try {
    contract_run(h, D, sweeps);
    trim_free_list(h);
    search_logz(h);
  } catch (...) {   // no block allocated by this call survives it: the handle is back at its pre-call footprint
    cudaStreamSynchronize(h->stream);
    mps_free(h);
    h->release_since(mark);
    trim_free_list(h);
    throw;
  }
  trim_free_list(h);
  TN_API_END
}

int tn_log_z(tn_handle* h, double* log_z) {
  TN_API_BEGIN
  if (!h || !log_z) tn_throw(TN_ERR_ARG, "NULL argument");
  if (!h->have_mps || !h->have_logz) tn_throw(TN_ERR_STATE, "tn_log_z before tn_contract");
  *log_z = h->log_z;
  TN_API_END
}

int tn_row_lognorm(tn_handle* h, int32_t y, double* lognorm) {
  TN_API_BEGIN
  if (!h || !lognorm) tn_throw(TN_ERR_ARG, "NULL argument");
  if (!h->have_mps) tn_throw(TN_ERR_STATE, "tn_row_lognorm before tn_contract");
  if (y < 1 || y > h->Ly) tn_throw(TN_ERR_ARG, "row out of range");
  *lognorm = h->lognorm[y];
  TN_API_END
}

int tn_mps_shape(tn_handle* h, int32_t y, int32_t j, int32_t* n_pos, int32_t* dl, int32_t* p, int32_t* dr) {
  TN_API_BEGIN
  if (!h) tn_throw(TN_ERR_ARG, "NULL argument");
  if (!h->have_mps) tn_throw(TN_ERR_STATE, "tn_mps_shape before tn_contract");
  if (y < 1 || y > h->Ly || j < 0 || j >= (int)h->rows[y].size()) tn_throw(TN_ERR_ARG, "index out of range");
  const MpsTensor& t = h->rows[y][j];
  if (n_pos) *n_pos = (int)h->rows[y].size();
  if (dl) *dl = t.dl;
  if (p) *p = t.p;
  if (dr) *dr = t.dr;
  TN_API_END
}

int tn_mps_tensor(tn_handle* h, int32_t y, int32_t j, double* out) {
  TN_API_BEGIN
  if (!h || !out) tn_throw(TN_ERR_ARG, "NULL argument");
  if (!h->have_mps) tn_throw(TN_ERR_STATE, "tn_mps_tensor before tn_contract");
  if (y < 1 || y > h->Ly || j < 0 || j >= (int)h->rows[y].size()) tn_throw(TN_ERR_ARG, "index out of range");
  const MpsTensor& t = h->rows[y][j];
  DeviceGuard dg(h);
  TN_CUDA(cudaMemcpyAsync(out, t.d, sizeof(double) * t.dl * t.p * t.dr, cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaStreamSynchronize(h->stream));
  TN_API_END
}

int tn_branch_and_bound(tn_handle* h, int32_t M, int32_t* n_out, int8_t* states, double* energies, double* logp,
                        double* log_pd) {
  TN_API_BEGIN
  if (!h || !n_out || !states || !energies || !logp) tn_throw(TN_ERR_ARG, "NULL argument");
  if (M < 1 || M > (1 << 20)) tn_throw(TN_ERR_ARG, "M must be in 1..2^20");
  if (!h->have_mps) tn_throw(TN_ERR_STATE, "tn_branch_and_bound before tn_contract");
  DeviceGuard dg(h);
  const unsigned long long mark = h->serial;
  try {
    search_run(h, M, n_out, states, energies, logp, log_pd);
  } catch (...) {
    cudaStreamSynchronize(h->stream);
    h->release_since(mark);
    trim_free_list(h);
    throw;
  }
  trim_free_list(h);
  TN_API_END
}

int tn_droplets(tn_handle* h, int32_t rank, int32_t* n, double* dE, int8_t* flips) {
  TN_API_BEGIN
  if (!h || !n) tn_throw(TN_ERR_ARG, "NULL argument");
  if (h->drop_K == 0) tn_throw(TN_ERR_STATE, "tn_droplets: the last tn_branch_and_bound did not run with TN_OPT_MERGE and TN_OPT_DROPLETS");
  if (rank < 0 || rank >= (int)h->drop_cnt.size()) tn_throw(TN_ERR_ARG, "rank out of range");
  const int k = h->drop_cnt[rank];
  *n = k;
  if (dE) std::copy(h->drop_dE.begin() + (size_t)rank * h->drop_K, h->drop_dE.begin() + (size_t)rank * h->drop_K + k, dE);
  if (flips) std::copy(h->drop_flips.begin() + (size_t)rank * h->drop_K * h->n_spins,
                       h->drop_flips.begin() + ((size_t)rank * h->drop_K + k) * h->n_spins, flips);
  TN_API_END
}

int tn_energy(tn_handle* h, int32_t n, const int8_t* states, double* energies) {
  TN_API_BEGIN
  if (!h || !states || !energies || n < 0) tn_throw(TN_ERR_ARG, "bad argument");
  DeviceGuard dg(h);
  const unsigned long long mark = h->serial;
  try {
    energy_run(h, n, states, energies);
  } catch (...) {
    cudaStreamSynchronize(h->stream);
    h->release_since(mark);
    trim_free_list(h);
    throw;
  }
  trim_free_list(h);
  TN_API_END
}

int tn_kernel_check(tn_handle* h, int32_t op, int64_t m, int32_t n, int32_t k, const double* A, const double* B,
                    double* Cout) {
  TN_API_BEGIN
  if (!h || !A || !Cout || m < 1 || n < 1 || k < 1) tn_throw(TN_ERR_ARG, "bad argument");
  need_device();
  DeviceGuard dg(h);
  const unsigned long long mark = h->serial;
  try {
    kernel_check_run(h, op, m, n, k, A, B, Cout);
  } catch (...) {
    cudaStreamSynchronize(h->stream);
    h->release_since(mark);
    trim_free_list(h);
    throw;
  }
  trim_free_list(h);
  TN_API_END
}

int tn_kernel_bench(tn_handle* h, int32_t op, int64_t m, int32_t n, int64_t k, int32_t iters, double* ms_per_call) {
  TN_API_BEGIN
  if (!h || !ms_per_call || m < 1 || n < 1 || k < 1) tn_throw(TN_ERR_ARG, "bad argument");
  need_device();
  DeviceGuard dg(h);
  const unsigned long long mark = h->serial;
  try {
    kernel_bench_run(h, op, m, n, k, iters, ms_per_call);
  } catch (...) {
    cudaStreamSynchronize(h->stream);
    h->release_since(mark);
    trim_free_list(h);
    throw;
  }
  trim_free_list(h);
  TN_API_END
}

int tn_lbp(tn_handle* h, int32_t iterations) {
  TN_API_BEGIN
  if (!h) tn_throw(TN_ERR_ARG, "handle is NULL");
  if (!h->have_beta) tn_throw(TN_ERR_STATE, "tn_lbp before tn_set_beta");
  if (iterations < 0 || iterations > 100000) tn_throw(TN_ERR_ARG, "iterations must be in 0..100000");
  DeviceGuard dg(h);
  lbp_run(h, iterations);
  TN_API_END
}

int tn_lbp_message(tn_handle* h, int32_t y, int32_t x, int32_t leg, int32_t* n, double* nu) {
  TN_API_BEGIN
  if (!h || !n || !nu) tn_throw(TN_ERR_ARG, "NULL argument");
  DeviceGuard dg(h);
  lbp_message(h, y, x, leg, n, nu);
  TN_API_END
}

int tn_lbp_marginals(tn_handle* h, int32_t y, int32_t x, int64_t n, const uint32_t* cell_states, double* logp) {
  TN_API_BEGIN
  if (!h || n < 0 || (n > 0 && (!cell_states || !logp))) tn_throw(TN_ERR_ARG, "bad argument");
  DeviceGuard dg(h);
  const unsigned long long mark = h->serial;
  try {
    lbp_marginals(h, y, x, n, cell_states, logp);
  } catch (...) {
    cudaStreamSynchronize(h->stream);
    h->release_since(mark);
    trim_free_list(h);
    throw;
  }
  trim_free_list(h);
  TN_API_END
}

int tn_lbp_select(tn_handle* h, int32_t y, int32_t x, int32_t K, int32_t* n_out, uint32_t* cell_states, double* logp) {
  TN_API_BEGIN
  if (!h || !n_out || !cell_states || !logp) tn_throw(TN_ERR_ARG, "NULL argument");
  DeviceGuard dg(h);
  const unsigned long long mark = h->serial;
  try {
    lbp_select(h, y, x, K, n_out, cell_states, logp);
  } catch (...) {
    cudaStreamSynchronize(h->stream);
    h->release_since(mark);
    trim_free_list(h);
    throw;
  }
  trim_free_list(h);
  TN_API_END
}

int tn_gemm_t_static(void* cuda_stream, int64_t m, int32_t n, int64_t k, const double* dA, int64_t lda, const double* dB,
                     int64_t ldb, double* dC, int64_t ldc) {
  TN_API_BEGIN
  need_device();
  gemm_t_static_run(cuda_stream, m, n, k, dA, lda, dB, ldb, dC, ldc);
  TN_API_END
}

int tn_get_stats(tn_handle* h, tn_stats* out) {
  TN_API_BEGIN
  if (!h || !out) tn_throw(TN_ERR_ARG, "NULL argument");
  DeviceGuard dg(h);
  *out = h->st;
  out->bytes_device = h->bytes_held;
  if (h->d_cnt) {
    unsigned long long c[2] = {0, 0};
    TN_CUDA(cudaMemcpyAsync(c, h->d_cnt, sizeof(c), cudaMemcpyDeviceToHost, h->stream));
    TN_CUDA(cudaStreamSynchronize(h->stream));
    out->jacobi_calls = (int64_t)c[0];
    out->jacobi_sweeps = (int64_t)c[1];
  }
  TN_API_END
}

void tn_destroy(tn_handle* h) {
  if (!h) return;
  try {
    DeviceGuard dg(h);
    cudaStreamSynchronize(h->stream);
    mps_free(h);
    lbp_free(h);
    tables_destroy(h);
    for (void* p : {(void*)h->d_eu, (void*)h->d_ev, (void*)h->d_J, (void*)h->d_h, (void*)h->d_cell_of,
                    (void*)h->d_bit_of, (void*)h->d_cnt})
      if (p) h->dfree(p);
    trim_free_list(h);
    for (auto& l : h->live) raw_free(h, l);
    h->live.clear();
  } catch (...) {
  }
  delete h;
}

}  // extern "C"
