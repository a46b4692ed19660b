// Batched small-K FP64 tensor-core GEMM with a fused weight epilogue.
//
//   C(batch; i, j) = weight(batch, i, j) * sum_{k < K} A(batch; i, k) * B(batch; k, j),      K <= 64 (a bond dimension)
//
// This is the shape of the two "project -> batched D x D product -> Boltzmann factor" diagrams of Fig. 7
// once the cell weight is factorised: the Theta-core build (batch = MPO-bond state k, rows
// (x, b), K = old bond) and the search conditionals (batch = beam element, rows (b, c_lo), columns a, K = bond
// of R_{y+1}).  With K <= 64 each output costs <= 128 FLOP, i.e. <= 16 FLOP per byte written: the kernel is bound
// by the HBM WRITE of C, so the whole K extent of both operands is staged in shared memory once per CTA (no k
// pipeline), rows of A are gathered through the projector tables by a row-pointer functor, and all weights are
// applied in registers before the only global store.
//
//   AR: const double* operator()(int batch, int i)      -> pointer to the K contiguous doubles of row i
//   BE: double operator()(int batch, int k, int j)      -> element of B
//   EP: Row row(int batch, int i);  put(Row&, batch, j, v);  put2(Row&, batch, j, v0, v1) (columns j, j+1);
//       static constexpr bool kReduce: if set, collect(Row&, double&, unsigned&) after each row and
//       tile_done(batch, row_tile, sum, count) once per (batch, row tile) with the CTA-reduced values (fixed order)
#pragma once
#include "gemm.cuh"

// A_SHARED: the rows of A do not depend on the batch -> one CTA keeps its A tile in shared memory and walks
// over `bg` consecutive batches (cuts the L2 -> SM read traffic, which otherwise equals the write traffic).
// Every CTA also walks over all column tiles of its rows with the same A tile.
template <int KP, int NT, bool A_SHARED, class AR, class BE, class EP>
__global__ void __launch_bounds__(256, 2) k_bgemm(int batches, int bg, int M, int N, int K, AR ar, BE be, EP ep) {
  constexpr int BM = 128, BN = 8 * NT, LDA = smem_ld(KP), LDB = smem_ld(BN);
  extern __shared__ __align__(16) double bg_smem[];
  double* sA = bg_smem;
  double* sB = bg_smem + BM * LDA;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int m0 = blockIdx.y * BM;
  const int b0 = blockIdx.x * bg, b1 = min(batches, b0 + bg);
  __shared__ double s_rz[8];
  __shared__ unsigned s_rn[8];
  for (int batch = b0; batch < b1; batch++) {
    double tz = 0.0;     // EP::kReduce: per-thread sum / count collected by the epilogue rows of this batch
    unsigned tn = 0;
    if (!A_SHARED || batch == b0) {
      __syncthreads();
      for (int r = warp; r < BM; r += 8) {
        const int gi = m0 + r;
        const double* src = gi < M ? ar(batch, gi) : nullptr;
#pragma unroll
        for (int k = lane; k < KP; k += 32) sA[r * LDA + k] = (src && k < K) ? __ldg(src + k) : 0.0;
      }
    }
    for (int n0 = 0; n0 < N; n0 += BN) {
      __syncthreads();
      for (int idx = tid; idx < KP * BN; idx += 256) {
        const int k = idx / BN, j = idx % BN;
        sB[k * LDB + j] = (k < K && n0 + j < N) ? be(batch, k, n0 + j) : 0.0;
      }
      __syncthreads();
      double acc[2][NT][2];
#pragma unroll
      for (int i = 0; i < 2; i++)
#pragma unroll
        for (int j = 0; j < NT; j++) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll
      for (int kk = 0; kk < KP; kk += 4) {
        const double fa0 = sA[(16 * warp + (lane >> 2)) * LDA + kk + (lane & 3)];
        const double fa1 = sA[(16 * warp + 8 + (lane >> 2)) * LDA + kk + (lane & 3)];
        const double* brow = sB + (kk + (lane & 3)) * LDB + (lane >> 2);
#pragma unroll
        for (int j = 0; j < NT; j++) {
          const double fb = brow[8 * j];
          dmma884(acc[0][j][0], acc[0][j][1], fa0, fb);
          dmma884(acc[1][j][0], acc[1][j][1], fa1, fb);
        }
      }
#pragma unroll
      for (int i = 0; i < 2; i++) {
        const int row = m0 + 16 * warp + 8 * i + (lane >> 2);
        if (row < M) {
          typename EP::Row rc = ep.row(batch, row);
#pragma unroll
          for (int j = 0; j < NT; j++) {
            const int col = n0 + 8 * j + 2 * (lane & 3);
            if (col + 1 < N) ep.put2(rc, batch, col, acc[i][j][0], acc[i][j][1]);
            else if (col < N) ep.put(rc, batch, col, acc[i][j][0]);
          }
          if constexpr (EP::kReduce) ep.collect(rc, tz, tn);
        }
      }
    }
    if constexpr (EP::kReduce) {   // ordered CTA reduction of the epilogue sums -> one partial per (batch, row tile)
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        tz += __shfl_xor_sync(0xffffffffu, tz, o);
        tn += __shfl_xor_sync(0xffffffffu, tn, o);
      }
      __syncthreads();
      if (lane == 0) { s_rz[warp] = tz; s_rn[warp] = tn; }
      __syncthreads();
      if (tid == 0) {
        double z = 0.0;
        unsigned nn = 0;
        for (int w = 0; w < 8; w++) { z += s_rz[w]; nn += s_rn[w]; }
        ep.tile_done(batch, blockIdx.y, z, nn);
      }
    }
  }
}

// Pipelined variant for a batch-independent A and a B whose rows are contiguous in memory (Theta-core build):
// the B tile of batch i+1 is fetched with 16-byte cp.async into the second shared buffer while batch i is
// multiplied and stored, so the only exposed latencies are the first fetch and the barriers.
//   BR: const double* operator()(int batch, int k) -> pointer to the N contiguous doubles of row k of B (16-byte aligned)
//   WARPS: 8 (128 rows per CTA) or 4 (64 rows): the narrow CTA halves the shared-memory footprint, so that the K = 64,
//   N = 64 instantiation (configs[3]) fits two independent CTAs per SM instead of one (barriers decoupled)
//   NBUF: B buffers.  With 3 the fetch of batch i+1 lands in a buffer last read two batches ago, so the barrier between
//   the multiply and the epilogue is not needed and the warps of a CTA drift out of phase (stores overlap DMMAs).
template <int KP, int NT, int WARPS, int NBUF, class AR, class BR, class EP>
__global__ void __launch_bounds__(32 * WARPS) k_bgemm_pipe(int batches, int bg, int M, int N, int K, AR ar, BR br, EP ep) {
  constexpr int BM = 16 * WARPS, NTH = 32 * WARPS, BN = 8 * NT, LDA = smem_ld(KP), LDB = smem_ld(BN);
  extern __shared__ __align__(16) double bg_smem[];
  double* sA = bg_smem;
  double* sB = bg_smem + BM * LDA;            // NBUF buffers of KP * LDB
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int m0 = blockIdx.y * BM;
  const int b0 = blockIdx.x * bg, b1 = min(batches, b0 + bg);
  auto fetch = [&](int batch, int buf) {
    double* dst = sB + buf * (KP * LDB);
    constexpr int G = BN / 2;
    for (int idx = tid; idx < KP * G; idx += NTH) {
      const int k = idx / G, g2 = 2 * (idx % G);
      const int rem = k < K ? N - g2 : 0;
      const int bytes = rem >= 2 ? 16 : rem == 1 ? 8 : 0;
      const double* src = bytes ? br(batch, k) + g2 : br(batch, 0);
      unsigned sa = (unsigned)__cvta_generic_to_shared(dst + k * LDB + g2);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(src), "r"(bytes));
    }
    asm volatile("cp.async.commit_group;");
  };
  fetch(b0, 0);
  for (int r = warp; r < BM; r += WARPS) {
    const int gi = m0 + r;
    const double* src = gi < M ? ar(b0, gi) : nullptr;
#pragma unroll
    for (int k = lane; k < KP; k += 32) sA[r * LDA + k] = (src && k < K) ? __ldg(src + k) : 0.0;
  }
  for (int batch = b0; batch < b1; batch++) {
    const int buf = (batch - b0) % NBUF;
    if (batch + 1 < b1) {
      fetch(batch + 1, (buf + 1) % NBUF);
      asm volatile("cp.async.wait_group 1;");
    } else {
      asm volatile("cp.async.wait_group 0;");
    }
    __syncthreads();
    const double* sb = sB + buf * (KP * LDB);
    // the epilogue's row descriptors (output pointer + gathered weights) are requested BEFORE the multiply so that
    // their global-load latency hides behind the DMMAs (ncu: long-scoreboard stalls in the epilogue otherwise)
    const int row0 = m0 + 16 * warp + (lane >> 2), row1 = row0 + 8;
    typename EP::Row rc0 = ep.row(batch, row0 < M ? row0 : 0), rc1 = ep.row(batch, row1 < M ? row1 : 0);
    double acc[2][NT][2];
#pragma unroll
    for (int i = 0; i < 2; i++)
#pragma unroll
      for (int j = 0; j < NT; j++) acc[i][j][0] = acc[i][j][1] = 0.0;
#pragma unroll
    for (int kk = 0; kk < KP; kk += 4) {
      const double fa0 = sA[(16 * warp + (lane >> 2)) * LDA + kk + (lane & 3)];
      const double fa1 = sA[(16 * warp + 8 + (lane >> 2)) * LDA + kk + (lane & 3)];
      const double* brow = sb + (kk + (lane & 3)) * LDB + (lane >> 2);
#pragma unroll
      for (int j = 0; j < NT; j++) {
        const double fb = brow[8 * j];
        dmma884(acc[0][j][0], acc[0][j][1], fa0, fb);
        dmma884(acc[1][j][0], acc[1][j][1], fa1, fb);
      }
    }
    if (NBUF < 3) __syncthreads();   // everyone is done with sb before the fetch of batch + 2 overwrites it
    if (row0 < M) {
#pragma unroll
      for (int j = 0; j < NT; j++) {
        const int col = 8 * j + 2 * (lane & 3);
        if (col + 1 < N) ep.put2(rc0, batch, col, acc[0][j][0], acc[0][j][1]);
        else if (col < N) ep.put(rc0, batch, col, acc[0][j][0]);
      }
    }
    if (row1 < M) {
#pragma unroll
      for (int j = 0; j < NT; j++) {
        const int col = 8 * j + 2 * (lane & 3);
        if (col + 1 < N) ep.put2(rc1, batch, col, acc[1][j][0], acc[1][j][1]);
        else if (col < N) ep.put(rc1, batch, col, acc[1][j][0]);
      }
    }
  }
}

template <int KP, int NT, class AR, class BR, class EP>
void launch_bgemm_pipe_knt(tn_handle* h, int batches, int M, int N, int K, const AR& ar, const BR& br, const EP& ep) {
  constexpr int WARPS = (KP * NT >= 64 * 8) ? 4 : 8;     // the largest tile takes the narrow CTA (two per SM)
  constexpr int BM = 16 * WARPS, BN = 8 * NT, LDA = smem_ld(KP), LDB = smem_ld(BN);
  constexpr int smem3 = (int)sizeof(double) * (BM * LDA + 3 * KP * LDB);
  constexpr int NBUF = smem3 <= 75 * 1024 ? 3 : 2;       // a third buffer only where three CTAs per SM still fit
  constexpr int smem = (int)sizeof(double) * (BM * LDA + NBUF * KP * LDB);
  TN_SMEM_OPT_IN(h, (k_bgemm_pipe<KP, NT, WARPS, NBUF, AR, BR, EP>), smem);
  const int mt = (M + BM - 1) / BM;
  const int bg = (int)std::max<i64>(1, std::min<i64>(16, (i64)batches * mt / (8 * (i64)h->sms)));
  dim3 grid((unsigned)((batches + bg - 1) / bg), (unsigned)mt);
  k_bgemm_pipe<KP, NT, WARPS, NBUF, AR, BR, EP><<<grid, 32 * WARPS, smem, h->stream>>>(batches, bg, M, N, K, ar, br, ep);
  h->st.kernel_launches++;
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) tn_throw(TN_ERR_CUDA, "k_bgemm_pipe launch failed: %s", cudaGetErrorString(e));
}

// K <= 64, N <= 64 and even (16-byte rows); returns false otherwise.
template <class AR, class BR, class EP>
bool launch_bgemm_pipe(tn_handle* h, int batches, int M, int N, int K, const AR& ar, const BR& br, const EP& ep) {
  if (K < 1 || K > 64 || N < 2 || N > 64 || (N & 1) || batches < 1 || M < 1 || (M + 63) / 64 > 65535) return false;
#define TN_PIPE_N(KP_)                                                                   \
  do {                                                                                   \
    if (N <= 16) launch_bgemm_pipe_knt<KP_, 2>(h, batches, M, N, K, ar, br, ep);         \
    else if (N <= 32) launch_bgemm_pipe_knt<KP_, 4>(h, batches, M, N, K, ar, br, ep);    \
    else launch_bgemm_pipe_knt<KP_, 8>(h, batches, M, N, K, ar, br, ep);                 \
  } while (0)
  if (K <= 16) TN_PIPE_N(16);
  else if (K <= 32) TN_PIPE_N(32);
  else if (K <= 48) TN_PIPE_N(48);
  else TN_PIPE_N(64);
#undef TN_PIPE_N
  return true;
}

template <int KP, int NT, bool A_SHARED, class AR, class BE, class EP>
void launch_bgemm_knt(tn_handle* h, int batches, int M, int N, int K, const AR& ar, const BE& be, const EP& ep) {
  constexpr int BM = 128, BN = 8 * NT, LDA = smem_ld(KP), LDB = smem_ld(BN);
  constexpr int smem = (int)sizeof(double) * (BM * LDA + KP * LDB);
  TN_SMEM_OPT_IN(h, (k_bgemm<KP, NT, A_SHARED, AR, BE, EP>), smem);
  const int mt = (M + BM - 1) / BM;
  int bg = 1;
  if (A_SHARED) {   // as many batches per CTA as still leave >= 4 waves of CTAs
    bg = (int)std::max<i64>(1, std::min<i64>(16, (i64)batches * mt / (8 * (i64)h->sms)));
  }
  dim3 grid((unsigned)((batches + bg - 1) / bg), (unsigned)mt);
  k_bgemm<KP, NT, A_SHARED, AR, BE, EP><<<grid, 256, smem, h->stream>>>(batches, bg, M, N, K, ar, be, ep);
  h->st.kernel_launches++;
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) tn_throw(TN_ERR_CUDA, "k_bgemm launch failed: %s", cudaGetErrorString(e));
}

template <int KP, bool A_SHARED, class AR, class BE, class EP>
void launch_bgemm_k(tn_handle* h, int batches, int M, int N, int K, const AR& ar, const BE& be, const EP& ep) {
  if (N <= 16) launch_bgemm_knt<KP, 2, A_SHARED>(h, batches, M, N, K, ar, be, ep);
  else if (N <= 32) launch_bgemm_knt<KP, 4, A_SHARED>(h, batches, M, N, K, ar, be, ep);
  else launch_bgemm_knt<KP, 8, A_SHARED>(h, batches, M, N, K, ar, be, ep);
}

// K <= 64 only (returns false otherwise: the caller keeps its generic k_gemm path for exact-mode bonds).
template <bool A_SHARED, class AR, class BE, class EP>
bool launch_bgemm(tn_handle* h, int batches, int M, int N, int K, const AR& ar, const BE& be, const EP& ep) {
  if (K < 1 || K > 64 || batches < 1 || M < 1 || N < 1 || (M + 127) / 128 > 65535) return false;
  if (K <= 16) launch_bgemm_k<16, A_SHARED>(h, batches, M, N, K, ar, be, ep);
  else if (K <= 32) launch_bgemm_k<32, A_SHARED>(h, batches, M, N, K, ar, be, ep);
  else if (K <= 48) launch_bgemm_k<48, A_SHARED>(h, batches, M, N, K, ar, be, ep);
  else launch_bgemm_k<64, A_SHARED>(h, batches, M, N, K, ar, be, ep);
  return true;
}
