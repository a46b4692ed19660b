// Streaming tall x skinny FP64 tensor-core GEMMs: the "Theta-core x skinny" applies of a2/a3 (Fig. 7
// the O(chi^3 d) batched products are, with the explicit Theta-core, plain GEMMs with one
// huge operand read once from HBM and a skinny operand of <= 96 columns).
//
//   N:  C[M x N] = A[M x K]   . B[K x N]      A row-major (lda), streamed by row blocks
//   T:  C[K x N] = A[M x K]^T . B[M x N]      A row-major (lda), streamed by column blocks, reduced over rows
//
// Both: N <= 96 (all columns in one CTA), operands move global -> shared with 16-byte cp.async in a 3-stage
// ring (zero-filled at the ragged edges), fragments for mma.sync.m8n8k4.f64 (SASS DMMA) are read from
// shared memory with conflict-free strides (== 4 mod 16 doubles), 8 warps x (16 rows x N) register tiles.
// Arithmetic intensity is N/4 FLOP/B, so the kernel is DMMA-bound for N >= 24 and HBM-bound below.
// Small row counts use narrower CTAs and a split over the reduction (ordered workspace reduce: deterministic).
#include "kernels.cuh"

namespace {

constexpr int TS_BK = 16, TS_STAGES = 3;

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

// TRANS = false: CTA owns rows [m0, m0+BM) of A / C, reduction index = columns of A.
// TRANS = true : CTA owns columns [m0, m0+BM) of A (= rows of C), reduction index = rows of A.
// In both cases "i" is the output row (BM per CTA, 8 RPW per warp) and "kk" the reduction index.
// RPW = 8-row fragments per warp: 2 (16 rows) by default; 3 (24 rows per warp, 192 per CTA) for narrow column counts,
// where the multiply is limited by the shared-memory fragment loads per DMMA (measured: 74 % of the DMMA peak at 48
// columns against 86 % at 80): 3 NT DMMAs per 3 + NT fragment loads instead of 2 NT per 2 + NT, still two CTAs per SM.
template <int NT, int WARPS, bool TRANS, int RPW = 2>
__global__ void __launch_bounds__(WARPS * 32, (NT <= 10 || WARPS < 8) ? 2 : 1)
k_tsgemm(const double* __restrict__ A, i64 lda, const double* __restrict__ B, i64 ldb, double* __restrict__ C, i64 ldc,
         i64 Mout, int Nfull, i64 Kred, i64 kper, double* __restrict__ ws, int nz, i64 sBz, i64 sCz) {
  constexpr int BM = 8 * RPW * WARPS, NTH = 32 * WARPS, NP = 8 * NT;
  constexpr int LDA = TRANS ? smem_ld(BM) : smem_ld(TS_BK);   // doubles
  constexpr int LDB = smem_ld(NP);
  constexpr int A_ELEMS = TRANS ? TS_BK * LDA : BM * LDA;
  constexpr int B_ELEMS = TS_BK * LDB;
  extern __shared__ __align__(16) double smem[];
  double* sA = smem;
  double* sB = smem + TS_STAGES * A_ELEMS;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const i64 m0 = (i64)blockIdx.x * BM;
  const int split = blockIdx.y, nsplit = gridDim.y;
  const int bz = blockIdx.z / nz;                    // batch (A shared, B and C strided)
  const int n_off = (blockIdx.z % nz) * NP;          // column chunk (N > 96 is cut into chunks of NP columns)
  const int N = min(NP, Nfull - n_off);
  B += n_off + (i64)bz * sBz;
  const i64 k0 = (i64)split * kper, k1 = min(Kred, k0 + kper);
  const int nkt = k1 > k0 ? (int)((k1 - k0 + TS_BK - 1) / TS_BK) : 0;

  auto load_stage = [&](int stage, int kt) {
    const i64 kb = k0 + (i64)kt * TS_BK;
    double* a = sA + stage * A_ELEMS;
    double* b = sB + stage * B_ELEMS;
    if (!TRANS) {
      constexpr int G = TS_BK / 2;                      // 16-byte granules per row
      for (int idx = tid; idx < BM * G; idx += NTH) {
        const int r = idx / G, g = idx % G;
        const i64 gr = m0 + r, gk = kb + 2 * g;
        i64 rem = gr < Mout ? (k1 - gk) : 0;
        int bytes = rem >= 2 ? 16 : rem == 1 ? 8 : 0;
        const double* src = bytes ? A + gr * lda + gk : A;
        cp_async16(a + r * LDA + 2 * g, src, bytes);
      }
    } else {
      constexpr int G = BM / 2;
      for (int idx = tid; idx < TS_BK * G; idx += NTH) {
        const int r = idx / G, g = idx % G;
        const i64 gk = kb + r, gc = m0 + 2 * g;
        i64 rem = gk < k1 ? (Mout - gc) : 0;
        int bytes = rem >= 2 ? 16 : rem == 1 ? 8 : 0;
        const double* src = bytes ? A + gk * lda + gc : A;
        cp_async16(a + r * LDA + 2 * g, src, bytes);
      }
    }
    {
      constexpr int G = NP / 2;
      for (int idx = tid; idx < TS_BK * G; idx += NTH) {
        const int r = idx / G, g = idx % G;
        const i64 gk = kb + r;
        const int gc = 2 * g;
        int rem = gk < k1 ? (N - gc) : 0;
        int bytes = rem >= 2 ? 16 : rem == 1 ? 8 : 0;
        const double* src = bytes ? B + gk * ldb + gc : B;
        cp_async16(b + r * LDB + 2 * g, src, bytes);
      }
    }
  };

  double acc[RPW][NT][2];
#pragma unroll
  for (int i = 0; i < RPW; i++)
#pragma unroll
    for (int j = 0; j < NT; j++) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
  for (int s = 0; s < TS_STAGES - 1; s++) {
    if (s < nkt) load_stage(s, s);
    cp_async_commit();
  }
  for (int kt = 0; kt < nkt; kt++) {
    cp_async_wait<TS_STAGES - 2>();
    __syncthreads();
    if (kt + TS_STAGES - 1 < nkt) load_stage((kt + TS_STAGES - 1) % TS_STAGES, kt + TS_STAGES - 1);
    cp_async_commit();
    const double* a = sA + (kt % TS_STAGES) * A_ELEMS;
    const double* b = sB + (kt % TS_STAGES) * B_ELEMS;
#pragma unroll
    for (int kk = 0; kk < TS_BK; kk += 4) {
      double fa[RPW];
#pragma unroll
      for (int i = 0; i < RPW; i++)
        fa[i] = TRANS ? a[(kk + (lane & 3)) * LDA + 8 * RPW * warp + 8 * i + (lane >> 2)]
                      : a[(8 * RPW * warp + 8 * i + (lane >> 2)) * LDA + kk + (lane & 3)];
      const double* brow = b + (kk + (lane & 3)) * LDB + (lane >> 2);
#pragma unroll
      for (int j = 0; j < NT; j++) {
        const double fb = brow[8 * j];
#pragma unroll
        for (int i = 0; i < RPW; i++) dmma884(acc[i][j][0], acc[i][j][1], fa[i], fb);
      }
    }
  }
  cp_async_wait<0>();
  // ---- epilogue
  double* out = (nsplit > 1 ? ws + ((size_t)bz * nsplit + split) * Mout * Nfull : C + (i64)bz * sCz) + n_off;
  const i64 ldo = nsplit > 1 ? Nfull : ldc;
#pragma unroll
  for (int i = 0; i < RPW; i++) {
    const i64 row = m0 + 8 * RPW * warp + 8 * i + (lane >> 2);
    if (row < Mout) {
#pragma unroll
      for (int j = 0; j < NT; j++) {
        const int col = 8 * j + 2 * (lane & 3);
        if (col < N) out[row * ldo + col] = acc[i][j][0];
        if (col + 1 < N) out[row * ldo + col + 1] = acc[i][j][1];
      }
    }
  }
}

// C[i][j] = sum_s ws[s][i][j]  (fixed order)
__global__ void k_ts_reduce(const double* __restrict__ ws, int nsplit, i64 M, int N, double* __restrict__ C, i64 ldc,
                            i64 sCz) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= M * N) return;
  const int bz = blockIdx.y;
  double s = 0.0;
  for (int sp = 0; sp < nsplit; sp++) s += ws[((size_t)bz * nsplit + sp) * M * N + t];
  C[(i64)bz * sCz + (t / N) * ldc + t % N] = s;
}

struct TsBatch { int n = 1; i64 sB = 0, sC = 0; };   // independent products sharing A: B_z = B + z sB, C_z = C + z sC

template <int NT, int WARPS, bool TRANS, int RPW = 2>
void launch_ts(tn_handle* h, const double* A, i64 lda, const double* B, i64 ldb, double* C, i64 ldc, i64 Mout, int N,
               i64 Kred, int nsplit, const TsBatch& tsb) {
  constexpr int BM = 8 * RPW * WARPS, NP = 8 * NT;
  constexpr int LDA = TRANS ? smem_ld(BM) : smem_ld(TS_BK), LDB = smem_ld(NP);
  constexpr size_t smem = sizeof(double) * TS_STAGES * ((TRANS ? TS_BK * LDA : BM * LDA) + TS_BK * LDB);
  TN_SMEM_OPT_IN(h, (k_tsgemm<NT, WARPS, TRANS, RPW>), smem);
  i64 kper = ((Kred + nsplit - 1) / nsplit + TS_BK - 1) / TS_BK * TS_BK;
  nsplit = (int)((Kred + kper - 1) / kper);
  const int nbz = tsb.n, nz = (N + NP - 1) / NP;
  double* ws = nsplit > 1 ? h->dalloc<double>((size_t)nbz * nsplit * Mout * N) : nullptr;
  dim3 grid((unsigned)((Mout + BM - 1) / BM), (unsigned)nsplit, (unsigned)(nz * nbz));
  k_tsgemm<NT, WARPS, TRANS, RPW><<<grid, WARPS * 32, smem, h->stream>>>(A, lda, B, ldb, C, ldc, Mout, N, Kred, kper, ws, nz,
                                                                          tsb.sB, tsb.sC);
  TN_LAUNCH_CHECK(h);
  if (nsplit > 1) {
    k_ts_reduce<<<dim3(cdiv(Mout * N, 256), nbz), 256, 0, h->stream>>>(ws, nsplit, Mout, N, C, ldc, tsb.sC);
    TN_LAUNCH_CHECK(h);
    h->dfree(ws);
  }
}

// CTA width and reduction split: minimise  waves x (per-CTA work + fixed cost) + split-workspace traffic.
// Measured on B200 (profiles/): wide CTAs win everywhere; the split mostly repairs wave quantisation when the
// output has fewer row blocks than 2 CTA slots per SM.
template <int NT, bool TRANS>
void pick_warps(tn_handle* h, const double* A, i64 lda, const double* B, i64 ldb, double* C, i64 ldc, i64 Mout, int N,
                i64 Kred, const TsBatch& tsb) {
  int warps = Mout > 64 ? 8 : Mout > 32 ? 4 : 2;
  // 24 rows per warp for 40..48 columns once the output has enough rows to fill the GPU with the 192-row tiles
  // (measured on B200: 74 -> 80 % of the DMMA peak at 48 columns; neutral at 40, worse at 24, so only NT = 5, 6)
  constexpr bool kWide = NT >= 5 && NT <= 6;
  const bool enough = !TRANS && Mout >= (i64)192 * 2 * h->sms;   // (the T variant loses more to its split quantisation: 75 -> 71 %)
  const int rpw = (kWide && warps == 8 && h->ts_rpw3 && enough) ? 3 : 2;
  const int bm = 8 * rpw * warps;
  const i64 tiles = (Mout + bm - 1) / bm * ((N + 8 * NT - 1) / (8 * NT)) * tsb.n;
  const int slots = h->sms * ((NT <= 10 || warps < 8) ? 2 : 1);
  const double t_k = 2.0 * bm * (8 * NT) * slots / 37e12;              // seconds per reduction index per CTA
  const double t_ws = (double)Mout * N * 16.0 / 6e12 + 2e-7;           // seconds per extra split (write + read)
  int best = 1;
  double best_t = 1e30;
  const int smax = (int)std::max<i64>(1, std::min<i64>(64, Kred / 128));
  for (int sp = 1; sp <= smax; sp++) {
    const i64 waves = (tiles * sp + slots - 1) / slots;
    const double t = waves * ((double)((Kred + sp - 1) / sp) + 96.0) * t_k + (sp > 1 ? sp * t_ws + 6e-6 : 0.0);
    if (t < best_t) { best_t = t; best = sp; }
  }
  if constexpr (kWide) {
    if (rpw == 3) { launch_ts<NT, 8, TRANS, 3>(h, A, lda, B, ldb, C, ldc, Mout, N, Kred, best, tsb); return; }
  }
  if (warps == 8) launch_ts<NT, 8, TRANS>(h, A, lda, B, ldb, C, ldc, Mout, N, Kred, best, tsb);
  else if (warps == 4) launch_ts<NT, 4, TRANS>(h, A, lda, B, ldb, C, ldc, Mout, N, Kred, best, tsb);
  else launch_ts<NT, 2, TRANS>(h, A, lda, B, ldb, C, ldc, Mout, N, Kred, best, tsb);
}

template <bool TRANS>
void pick_nt(tn_handle* h, const double* A, i64 lda, const double* B, i64 ldb, double* C, i64 ldc, i64 Mout, int N,
             i64 Kred, const TsBatch& tsb) {
  if (N > 96) { pick_warps<8, TRANS>(h, A, lda, B, ldb, C, ldc, Mout, N, Kred, tsb); return; }   // chunks of 64 columns
  switch ((N + 7) / 8) {   // one 8-column register tile per 8 columns: no padding beyond the last tile
#define TN_TS_CASE(NT_) case NT_: pick_warps<NT_, TRANS>(h, A, lda, B, ldb, C, ldc, Mout, N, Kred, tsb); break;
    TN_TS_CASE(1) TN_TS_CASE(2) TN_TS_CASE(3) TN_TS_CASE(4) TN_TS_CASE(5) TN_TS_CASE(6)
    TN_TS_CASE(7) TN_TS_CASE(8) TN_TS_CASE(9) TN_TS_CASE(10) TN_TS_CASE(11) TN_TS_CASE(12)
#undef TN_TS_CASE
    default: break;
  }
}

bool aligned16(const void* p) { return ((uintptr_t)p & 15) == 0; }

}  // namespace

static bool tsgemm_impl(tn_handle* h, bool trans, i64 M, int N, i64 K, const double* A, i64 lda, const double* B, i64 ldb,
                        double* C, i64 ldc, const TsBatch& tsb) {
  if (N < 1 || M < 1 || K < 1) return false;
  if ((lda & 1) || (ldb & 1) || !aligned16(A) || !aligned16(B)) return false;
  if (trans) pick_nt<true>(h, A, lda, B, ldb, C, ldc, K, N, M, tsb);    // output rows = K (columns of A), reduce over M
  else pick_nt<false>(h, A, lda, B, ldb, C, ldc, M, N, K, tsb);
  return true;
}

// Returns false when the shapes / alignment do not fit (the caller falls back to the generic k_gemm).
bool tsgemm(tn_handle* h, bool trans, i64 M, int N, i64 K, const double* A, i64 lda, const double* B, i64 ldb, double* C,
            i64 ldc) {
  return tsgemm_impl(h, trans, M, N, K, A, lda, B, ldb, C, ldc, TsBatch());
}

// nbatch independent products with a shared A: B_z = B + z sB, C_z = C + z sC.
bool tsgemm_batched(tn_handle* h, bool trans, i64 M, int N, i64 K, const double* A, i64 lda, const double* B, i64 ldb,
                    i64 sB, double* C, i64 ldc, i64 sC, int nbatch) {
  if (nbatch < 1 || nbatch > 16384 || (sB & 1)) return false;
  TsBatch tsb;
  tsb.n = nbatch; tsb.sB = sB; tsb.sC = sC;
  return tsgemm_impl(h, trans, M, N, K, A, lda, B, ldb, C, ldc, tsb);
}

// =====================================================================================================================
// Allocation-free entry point (tn_gemm_t_static, include/tn.h): C[k x n] = A[m x k]^T . B[m x n], the "Theta-core^T x
// skinny" apply with its split-over-the-reduction workspace in a file-scope device array instead of a device allocation:
// for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it).
//   * The scratch is TN_STATIC_SCRATCH_DOUBLES doubles (8 MiB); every GPU that loads the library holds it until exit.
//   * In HOST code the array's name is a host-side stand-in, not a device address: its device address is looked up once per
//     device, with that device current, by cudaGetSymbolAddress below, and that pointer is what the kernels get.
//   * Every call shares the array and it keeps the last call's contents.  Nothing has to start at zero: every workspace
//     entry the reduction reads is written first by the GEMM kernel of the same call (each split CTA stores its whole
//     in-range tile, zero or not).  Calls that overlap on the GPU (different streams, or graph branches) RACE on it.
//   * No cudaMalloc / cudaFree / allocating library routine, no synchronisation: two kernels are queued on the stream.
// =====================================================================================================================
static constexpr size_t TN_STATIC_SCRATCH_DOUBLES = (size_t)1 << 20;
static __device__ __align__(256) double g_ts_static_scratch[TN_STATIC_SCRATCH_DOUBLES];

namespace {

struct DevOnly { int device; };   // what TN_SMEM_OPT_IN needs from a handle

template <int NT>
void launch_ts_static(int dev, cudaStream_t st, const double* A, i64 lda, const double* B, i64 ldb, double* C, i64 ldc,
                      i64 Mout, int N, i64 Kred, int nsplit, double* scratch) {
  constexpr int WARPS = 8, BM = 16 * WARPS, NP = 8 * NT;
  constexpr int LDA = smem_ld(BM), LDB = smem_ld(NP);
  constexpr size_t smem = sizeof(double) * TS_STAGES * (TS_BK * LDA + TS_BK * LDB);
  DevOnly d{dev};
  TN_SMEM_OPT_IN(&d, (k_tsgemm<NT, WARPS, true>), smem);
  const i64 kper = ((Kred + nsplit - 1) / nsplit + TS_BK - 1) / TS_BK * TS_BK;
  nsplit = (int)((Kred + kper - 1) / kper);
  dim3 grid((unsigned)((Mout + BM - 1) / BM), (unsigned)nsplit, 1u);
  k_tsgemm<NT, WARPS, true><<<grid, WARPS * 32, smem, st>>>(A, lda, B, ldb, C, ldc, Mout, N, Kred, kper,
                                                           nsplit > 1 ? scratch : nullptr, 1, 0, 0);
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) tn_throw(TN_ERR_CUDA, "tn_gemm_t_static: launch failed: %s", cudaGetErrorString(e));
  if (nsplit > 1) {
    k_ts_reduce<<<dim3((unsigned)((Mout * N + 255) / 256), 1u), 256, 0, st>>>(scratch, nsplit, Mout, N, C, ldc, 0);
    e = cudaPeekAtLastError();
    if (e != cudaSuccess) tn_throw(TN_ERR_CUDA, "tn_gemm_t_static: reduce launch failed: %s", cudaGetErrorString(e));
  }
}

}  // namespace

void gemm_t_static_run(void* stream, i64 m, int n, i64 k, const double* A, i64 lda, const double* B, i64 ldb, double* C,
                       i64 ldc) {
  if (!A || !B || !C || m < 1 || n < 1 || k < 1) tn_throw(TN_ERR_ARG, "tn_gemm_t_static: NULL pointer or non-positive size");
  if (n > 96) tn_throw(TN_ERR_ARG, "tn_gemm_t_static: n = %d > 96 columns", n);
  if (lda < k || ldb < n || ldc < n || (lda & 1) || (ldb & 1) || !aligned16(A) || !aligned16(B))
    tn_throw(TN_ERR_ARG, "tn_gemm_t_static: lda >= k, ldb >= n, ldc >= n, lda and ldb even, A and B 16-byte aligned are required");
  if ((size_t)k * (size_t)n * 2 > TN_STATIC_SCRATCH_DOUBLES)
    tn_throw(TN_ERR_ARG, "tn_gemm_t_static: k * n = %lld exceeds the static scratch (two partial products of k * n doubles "
             "must fit %zu doubles = %zu MiB); use tn_kernel_check / the handle-based path for larger outputs",
             (long long)(k * n), TN_STATIC_SCRATCH_DOUBLES, TN_STATIC_SCRATCH_DOUBLES * sizeof(double) >> 20);
  int dev = 0;
  TN_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) tn_throw(TN_ERR_ARG, "tn_gemm_t_static: device ordinal %d not supported", dev);
  // set-up, once per device, with that device current: device address of the scratch array and the SM count
  static double* scratch_dev[64] = {nullptr};
  static int sms_dev[64] = {0};
  if (!scratch_dev[dev]) {
    double* p = nullptr;
    TN_CUDA(cudaGetSymbolAddress((void**)&p, g_ts_static_scratch));
    if (!p) tn_throw(TN_ERR_CUDA, "tn_gemm_t_static: cudaGetSymbolAddress returned NULL");
    TN_CUDA(cudaDeviceGetAttribute(&sms_dev[dev], cudaDevAttrMultiProcessorCount, dev));
    scratch_dev[dev] = p;
  }
  // split over the reduction (rows of A): enough CTAs for two waves, at least 128 rows per split, bounded by the scratch
  const i64 tiles = (k + 127) / 128;
  i64 want = (2 * (i64)sms_dev[dev] + tiles - 1) / tiles;
  want = std::min<i64>(want, std::max<i64>(1, m / 128));
  want = std::min<i64>(want, 64);
  want = std::min<i64>(want, (i64)(TN_STATIC_SCRATCH_DOUBLES / ((size_t)k * n)));
  const int nsplit = (int)std::max<i64>(1, want);
  cudaStream_t st = (cudaStream_t)stream;
  switch ((n + 7) / 8) {
#define TN_TS_CASE(NT_) case NT_: launch_ts_static<NT_>(dev, st, A, lda, B, ldb, C, ldc, k, n, m, nsplit, scratch_dev[dev]); break;
    TN_TS_CASE(1) TN_TS_CASE(2) TN_TS_CASE(3) TN_TS_CASE(4) TN_TS_CASE(5) TN_TS_CASE(6)
    TN_TS_CASE(7) TN_TS_CASE(8) TN_TS_CASE(9) TN_TS_CASE(10) TN_TS_CASE(11) TN_TS_CASE(12)
#undef TN_TS_CASE
    default: tn_throw(TN_ERR_ARG, "tn_gemm_t_static: n = %d", n);
  }
}
