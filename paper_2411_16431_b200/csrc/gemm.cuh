// FP64 tensor-core (DMMA m8n8k4) tile GEMM with functor loaders/epilogues.
// Every dense contraction of the path (Theta-core build, Theta x skinny applies, edge-matrix
// applies, Gram matrices, search GEMMs) is an instantiation of k_gemm with its own addressing.
// sm_100a has no tcgen05 kind for f64: FP64 tensor math is mma.sync DMMA (SASS DMMA.8x8x4),
// measured peak 37.2 TFLOP/s on this B200 (profiles/r01_fp64_peak.md).
#pragma once
#include "tn_common.cuh"

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

__host__ __device__ constexpr int smem_ld(int n) { return n + ((4 - n % 16) + 16) % 16; }  // == 4 (mod 16): conflict-free fragments

// C(batch; i, j) = sum_{k in split range} A(batch; i, k) * B(batch; k, j)
//   al(batch, i, k) -> double, bl(batch, k, j) -> double, ep(batch, split, i, j, acc)
//   grid: x = batch * nsplit, y = tile_m, z = tile_n.  A_KFAST / B_NFAST pick the loader's
//   fastest-running index so that global reads coalesce.
template <int BM, int BN, int BK, int WGM, int WGN, bool A_KFAST, bool B_NFAST, class AL, class BL, class EP>
__global__ void __launch_bounds__(WGM* WGN * 32) k_gemm(int M, int N, int K, int nsplit, AL al, BL bl, EP ep) {
  constexpr int NT = WGM * WGN * 32;
  constexpr int WM = BM / WGM, WN = BN / WGN;
  constexpr int TM = WM / 8, TN = WN / 8;
  constexpr int LDA = smem_ld(BM), LDB = smem_ld(BN);
  constexpr int AE = (BM * BK + NT - 1) / NT, BE = (BK * BN + NT - 1) / NT;
  static_assert(WM % 8 == 0 && WN % 8 == 0 && BK % 4 == 0, "tile shape");
  __shared__ double As[2][BK * LDA];
  __shared__ double Bs[2][BK * LDB];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / WGN) * WM, wn0 = (warp % WGN) * WN;
  const int batch = blockIdx.x / nsplit, split = blockIdx.x % nsplit;
  const int kper = (((K + nsplit - 1) / nsplit) + BK - 1) / BK * BK;
  const int k0 = split * kper, k1 = min(K, k0 + kper);
  const int m0 = blockIdx.y * BM, n0 = blockIdx.z * BN;

  double acc[TM][TN][2];
#pragma unroll
  for (int i = 0; i < TM; i++)
#pragma unroll
    for (int j = 0; j < TN; j++) acc[i][j][0] = acc[i][j][1] = 0.0;

  double ra[AE], rb[BE];
  auto gload = [&](int kb) {
#pragma unroll
    for (int e = 0; e < AE; e++) {
      int idx = tid + e * NT;
      int i = A_KFAST ? idx / BK : idx % BM, k = A_KFAST ? idx % BK : idx / BM;
      int gi = m0 + i, gk = kb + k;
      ra[e] = (idx < BM * BK && gi < M && gk < k1) ? al(batch, gi, gk) : 0.0;
    }
#pragma unroll
    for (int e = 0; e < BE; e++) {
      int idx = tid + e * NT;
      int k = B_NFAST ? idx / BN : idx % BK, j = B_NFAST ? idx % BN : idx / BK;
      int gk = kb + k, gj = n0 + j;
      rb[e] = (idx < BK * BN && gk < k1 && gj < N) ? bl(batch, gk, gj) : 0.0;
    }
  };
  auto sstore = [&](int buf) {
#pragma unroll
    for (int e = 0; e < AE; e++) {
      int idx = tid + e * NT;
      int i = A_KFAST ? idx / BK : idx % BM, k = A_KFAST ? idx % BK : idx / BM;
      if (idx < BM * BK) As[buf][k * LDA + i] = ra[e];
    }
#pragma unroll
    for (int e = 0; e < BE; e++) {
      int idx = tid + e * NT;
      int k = B_NFAST ? idx / BN : idx % BK, j = B_NFAST ? idx % BN : idx / BK;
      if (idx < BK * BN) Bs[buf][k * LDB + j] = rb[e];
    }
  };

  int buf = 0;
  if (k0 < k1) {
    gload(k0);
    sstore(0);
  }
  __syncthreads();
  for (int kb = k0; kb < k1; kb += BK) {
    const bool more = kb + BK < k1;
    if (more) gload(kb + BK);
    const double* as = As[buf];
    const double* bs = Bs[buf];
#pragma unroll
    for (int kk = 0; kk < BK; kk += 4) {
      double fa[TM], fb[TN];
#pragma unroll
      for (int i = 0; i < TM; i++) fa[i] = as[(kk + (lane & 3)) * LDA + wm0 + 8 * i + (lane >> 2)];
#pragma unroll
      for (int j = 0; j < TN; j++) fb[j] = bs[(kk + (lane & 3)) * LDB + wn0 + 8 * j + (lane >> 2)];
#pragma unroll
      for (int i = 0; i < TM; i++)
#pragma unroll
        for (int j = 0; j < TN; j++) dmma884(acc[i][j][0], acc[i][j][1], fa[i], fb[j]);
    }
    if (more) sstore(buf ^ 1);
    __syncthreads();
    buf ^= 1;
  }
#pragma unroll
  for (int i = 0; i < TM; i++)
#pragma unroll
    for (int j = 0; j < TN; j++) {
      int row = m0 + wm0 + 8 * i + (lane >> 2);
      int col = n0 + wn0 + 8 * j + 2 * (lane & 3);
      if (row < M) {
        if (col < N) ep(batch, split, row, col, acc[i][j][0]);
        if (col + 1 < N) ep(batch, split, row, col + 1, acc[i][j][1]);
      }
    }
}

// ---- general strided operands: two-level batch (b1, b2), element strides in doubles ----------
struct LdGen {
  const double* p;
  i64 sb1, sb2, s0, s1;   // s0: stride of the first matrix index, s1: of the second
  int B2;
  __device__ __forceinline__ double operator()(int batch, int i0, int i1) const {
    return __ldg(p + (i64)(batch / B2) * sb1 + (i64)(batch % B2) * sb2 + (i64)i0 * s0 + (i64)i1 * s1);
  }
};
struct StGen {
  double* p;
  i64 sb1, sb2, s0, s1;
  int B2;
  double alpha, beta;
  double* ws;   // split-K workspace [batch][split][M][N] when nsplit > 1
  int nsplit, M, N;
  __device__ __forceinline__ void operator()(int batch, int split, int i, int j, double v) const {
    if (nsplit > 1) {
      ws[(((i64)batch * nsplit + split) * M + i) * N + j] = v;
    } else {
      double* q = p + (i64)(batch / B2) * sb1 + (i64)(batch % B2) * sb2 + (i64)i * s0 + (i64)j * s1;
      *q = beta == 0.0 ? alpha * v : alpha * v + beta * *q;
    }
  }
};

struct GemmDesc {
  int M = 0, N = 0, K = 0;
  int B1 = 1, B2 = 1;
  const double* A = nullptr;
  i64 a_b1 = 0, a_b2 = 0, a_i = 0, a_k = 0;
  const double* B = nullptr;
  i64 b_b1 = 0, b_b2 = 0, b_k = 0, b_j = 0;
  double* C = nullptr;
  i64 c_b1 = 0, c_b2 = 0, c_i = 0, c_j = 0;
  double alpha = 1.0, beta = 0.0;
  int nsplit = 0;   // 0 = choose
};
// kernels.cu
void gemm_general(tn_handle* h, const GemmDesc& g);
// tsgemm.cu: streaming tall x skinny GEMM (N <= 96).  trans = false: C[M x N] = A[M x K] B[K x N];
// trans = true: C[K x N] = A[M x K]^T B[M x N].  Returns false if shape / alignment do not fit.
bool tsgemm(tn_handle* h, bool trans, i64 M, int N, i64 K, const double* A, i64 lda, const double* B, i64 ldb, double* C,
            i64 ldc);
bool tsgemm_batched(tn_handle* h, bool trans, i64 M, int N, i64 K, const double* A, i64 lda, const double* B, i64 ldb,
                    i64 sB, double* C, i64 ldc, i64 sC, int nbatch);
// plain row-major helpers: C[M,N] = op(A) op(B)
void gemm_rm(tn_handle* h, bool ta, bool tb, int M, int N, int K, const double* A, int lda, const double* B,
             int ldb, double* C, int ldc, double alpha = 1.0, double beta = 0.0);
