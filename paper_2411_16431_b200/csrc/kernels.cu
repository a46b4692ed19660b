// Shared device kernels: GEMM launchers, Jacobi, orthonormalisation, projector maps, Theta-core.
#include "kernels.cuh"
#include "bgemm.cuh"
#include <cstdarg>

// ============================================================================================
// generic strided GEMM launcher
// ============================================================================================
template <int BM, int BN, int WGM, int WGN, bool AK, bool BNF>
static void launch_gen(tn_handle* h, const GemmDesc& g, int nsplit, double* ws) {
  LdGen a{g.A, g.a_b1, g.a_b2, g.a_i, g.a_k, g.B2};
  LdGen b{g.B, g.b_b1, g.b_b2, g.b_k, g.b_j, g.B2};
  StGen c{g.C, g.c_b1, g.c_b2, g.c_i, g.c_j, g.B2, g.alpha, g.beta, ws, nsplit, g.M, g.N};
  dim3 grid((unsigned)(g.B1 * g.B2 * nsplit), (unsigned)cdiv(g.M, BM), (unsigned)cdiv(g.N, BN));
  k_gemm<BM, BN, 16, WGM, WGN, AK, BNF, LdGen, LdGen, StGen>
      <<<grid, WGM * WGN * 32, 0, h->stream>>>(g.M, g.N, g.K, nsplit, a, b, c);
  TN_LAUNCH_CHECK(h);
}

template <bool AK, bool BNF>
static void launch_gen_n(tn_handle* h, const GemmDesc& g, int nsplit, double* ws) {
  if (g.N <= 16) launch_gen<128, 16, 4, 1, AK, BNF>(h, g, nsplit, ws);
  else if (g.N <= 32) launch_gen<128, 32, 4, 1, AK, BNF>(h, g, nsplit, ws);
  else if (g.N <= 48) launch_gen<64, 48, 4, 1, AK, BNF>(h, g, nsplit, ws);
  else if (g.N <= 64) launch_gen<64, 64, 2, 2, AK, BNF>(h, g, nsplit, ws);
  else if (g.N <= 80) launch_gen<64, 80, 4, 1, AK, BNF>(h, g, nsplit, ws);
  else launch_gen<64, 64, 2, 2, AK, BNF>(h, g, nsplit, ws);
}

__global__ void k_splitk_reduce(const double* ws, int nsplit, int M, int N, StGen c, i64 total) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= total) return;
  int j = (int)(t % N);
  int i = (int)((t / N) % M);
  int batch = (int)(t / ((i64)M * N));
  double s = 0.0;
  for (int sp = 0; sp < nsplit; sp++) s += ws[(((i64)batch * nsplit + sp) * M + i) * N + j];
  c.nsplit = 1;
  c(batch, 0, i, j, s);
}

void gemm_general(tn_handle* h, const GemmDesc& g) {
  if (g.M <= 0 || g.N <= 0 || g.B1 * g.B2 <= 0) return;
  int nsplit = g.nsplit;
  const int bm = g.N <= 32 ? 128 : 64;
  const int bn = g.N <= 16 ? 16 : g.N <= 32 ? 32 : g.N <= 48 ? 48 : g.N <= 64 ? 64 : g.N <= 80 ? 80 : 64;
  if (nsplit <= 0) {
    i64 tiles = (i64)cdiv(g.M, bm) * cdiv(g.N, bn) * g.B1 * g.B2;
    nsplit = 1;
    if (tiles < h->sms && g.K >= 2048) {
      nsplit = (int)std::min<i64>((2 * h->sms + tiles - 1) / tiles, g.K / 512);
      if (nsplit < 1) nsplit = 1;
    }
  }
  double* ws = nullptr;
  if (nsplit > 1) ws = h->dalloc<double>((size_t)g.B1 * g.B2 * nsplit * g.M * g.N);
  const bool ak = (g.a_k == 1) || (g.a_i != 1 && g.a_k < g.a_i);
  const bool bnf = (g.b_j == 1) || (g.b_k != 1 && g.b_j < g.b_k);
  if (ak && bnf) launch_gen_n<true, true>(h, g, nsplit, ws);
  else if (ak && !bnf) launch_gen_n<true, false>(h, g, nsplit, ws);
  else if (!ak && bnf) launch_gen_n<false, true>(h, g, nsplit, ws);
  else launch_gen_n<false, false>(h, g, nsplit, ws);
  if (nsplit > 1) {
    StGen c{g.C, g.c_b1, g.c_b2, g.c_i, g.c_j, g.B2, g.alpha, g.beta, nullptr, 1, g.M, g.N};
    i64 total = (i64)g.B1 * g.B2 * g.M * g.N;
    k_splitk_reduce<<<cdiv(total, 256), 256, 0, h->stream>>>(ws, nsplit, g.M, g.N, c, total);
    TN_LAUNCH_CHECK(h);
    h->dfree(ws);
  }
}

// out[k][j] = in[j][k] (j < N), zero in the pad column
__global__ void k_transpose_pad(double* out, const double* in, int K, int N, int ldt, int ldb) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= K * ldt) return;
  int k = t / ldt, j = t % ldt;
  out[t] = j < N ? in[(i64)j * ldb + k] : 0.0;
}

void gemm_rm(tn_handle* h, bool ta, bool tb, int M, int N, int K, const double* A, int lda, const double* B,
             int ldb, double* C, int ldc, double alpha, double beta) {
  if (M <= 0 || N <= 0) return;
  if (alpha == 1.0 && beta == 0.0 && K > 0) {   // streaming cp.async kernel (tsgemm.cu)
    if (!tb) {
      if (!ta && tsgemm(h, false, M, N, K, A, lda, B, ldb, C, ldc)) return;
      if (ta && tsgemm(h, true, K, N, M, A, lda, B, ldb, C, ldc)) return;
    } else if ((i64)N * K <= 65536) {             // small B given transposed: transpose it first
      const int ldt = (N + 1) & ~1;
      DBuf<double> Bt(h, (size_t)K * ldt);
      k_transpose_pad<<<cdiv((i64)K * ldt, 256), 256, 0, h->stream>>>(Bt.p, B, K, N, ldt, ldb);
      TN_LAUNCH_CHECK(h);
      if (!ta && tsgemm(h, false, M, N, K, A, lda, Bt.p, ldt, C, ldc)) return;
      if (ta && tsgemm(h, true, K, N, M, A, lda, Bt.p, ldt, C, ldc)) return;
    }
  }
  GemmDesc g;
  g.M = M; g.N = N; g.K = K;
  g.A = A; g.a_i = ta ? 1 : lda; g.a_k = ta ? lda : 1;
  g.B = B; g.b_k = tb ? 1 : ldb; g.b_j = tb ? ldb : 1;
  g.C = C; g.c_i = ldc; g.c_j = 1;
  g.alpha = alpha; g.beta = beta;
  gemm_general(h, g);
}

// ============================================================================================
// small utilities
// ============================================================================================
__device__ __forceinline__ uint64_t mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
__global__ void k_fill_random(double* X, i64 n, uint64_t seed) {
  i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) X[i] = 2.0 * ((mix64(seed * 0x100000001B3ull + (uint64_t)i) >> 11) * (1.0 / 9007199254740992.0)) - 1.0;
}
// Omega[(p', gamma)][col] = uniform(-1,1) from the counter (seed, p', gamma, col): independent of any memory layout, so
// that the randomized SVD (TN_OPT_SVD_MODE = 1) draws the same block whatever the padding of the bonds
__global__ void k_fill_random_pgc(double* X, int pu, int g, int ks, uint64_t seed) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (i64)pu * g * ks) return;
  const uint64_t c = (uint64_t)(t % ks), gg = (uint64_t)((t / ks) % g), pp = (uint64_t)(t / ((i64)ks * g));
  const uint64_t ctr = seed * 0x100000001B3ull + ((pp * 4096ull + gg) * 1024ull + c);
  X[t] = 2.0 * ((mix64(ctr) >> 11) * (1.0 / 9007199254740992.0)) - 1.0;
}
void fill_random_pgc(tn_handle* h, double* X, int pu, int g, int ks, uint64_t seed) {
  const i64 n = (i64)pu * g * ks;
  if (n <= 0) return;
  k_fill_random_pgc<<<cdiv(n, 256), 256, 0, h->stream>>>(X, pu, g, ks, seed);
  TN_LAUNCH_CHECK(h);
}
void fill_random(tn_handle* h, double* X, i64 n, uint64_t seed) {
  if (n <= 0) return;
  k_fill_random<<<cdiv(n, 256), 256, 0, h->stream>>>(X, n, seed);
  TN_LAUNCH_CHECK(h);
}
__global__ void k_fill_value(double* X, i64 n, double v) {
  i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) X[i] = v;
}
void fill_value(tn_handle* h, double* X, i64 n, double v) {
  if (n <= 0) return;
  k_fill_value<<<cdiv(n, 256), 256, 0, h->stream>>>(X, n, v);
  TN_LAUNCH_CHECK(h);
}

__global__ void k_permute3(double* out, const double* in, int n0, int n1, int n2, i64 s0, i64 s1, i64 s2,
                           int mask_axis, const int* keep) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  i64 total = (i64)n0 * n1 * n2;
  if (t >= total) return;
  int i2 = (int)(t % n2), i1 = (int)((t / n2) % n1), i0 = (int)(t / ((i64)n1 * n2));
  double v = in[i0 * s0 + i1 * s1 + i2 * s2];
  if (mask_axis >= 0) {
    int idx = mask_axis == 0 ? i0 : mask_axis == 1 ? i1 : i2;
    if (idx >= *keep) v = 0.0;
  }
  out[t] = v;
}
void permute3(tn_handle* h, double* out, const double* in, int n0, int n1, int n2, i64 s0, i64 s1, i64 s2,
              int mask_axis, const int* keep) {
  i64 total = (i64)n0 * n1 * n2;
  if (total <= 0) return;
  k_permute3<<<cdiv(total, 256), 256, 0, h->stream>>>(out, in, n0, n1, n2, s0, s1, s2, mask_axis, keep);
  TN_LAUNCH_CHECK(h);
}

__global__ void k_scale_by(double* X, i64 n, const double* s, bool inverse) {
  i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) X[i] = inverse ? X[i] / *s : X[i] * *s;
}
void scale_by(tn_handle* h, double* X, i64 n, const double* s, bool inverse) {
  if (n <= 0) return;
  k_scale_by<<<cdiv(n, 256), 256, 0, h->stream>>>(X, n, s, inverse);
  TN_LAUNCH_CHECK(h);
}

__global__ void k_sumsq_part(const double* X, i64 n, double* part) {
  __shared__ double sh[256];
  double s = 0.0;
  for (i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (i64)gridDim.x * blockDim.x) s += X[i] * X[i];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) part[blockIdx.x] = sh[0];
}
__global__ void k_sumsq_final(const double* part, int np, double* out) {
  __shared__ double sh[256];
  double s = 0.0;
  for (int i = threadIdx.x; i < np; i += 256) s += part[i];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) *out = sqrt(sh[0]);
}
void frob_norm(tn_handle* h, const double* X, i64 n, double* out) {
  int nb = (int)std::min<i64>(592, std::max<i64>(1, (n + 255) / 256));
  double* part = h->dalloc<double>(nb);
  k_sumsq_part<<<nb, 256, 0, h->stream>>>(X, n, part);
  TN_LAUNCH_CHECK(h);
  k_sumsq_final<<<1, 256, 0, h->stream>>>(part, nb, out);
  TN_LAUNCH_CHECK(h);
  h->dfree(part);
}

// ============================================================================================
// one-sided Jacobi on rows (single CTA; working set in shared memory when it fits)
// ============================================================================================
// Working storage: Mw [c x r] (ldm), Ww [c x c].  Round-robin pair ordering; each warp owns a pair.
__device__ __forceinline__ double rcp_fast(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  y = y * (2.0 - x * y);
  return y * (2.0 - x * y);
}
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double hx = 0.5 * x;
  y = y * (1.5 - hx * y * y);
  return y * (1.5 - hx * y * y);
}
__global__ void __launch_bounds__(1024) k_jacobi_rows(const double* Min, int ld, int c, int r, double* Mout,
                                                      double* Wt, double* sig, double* gwork, int use_smem,
                                                      unsigned long long* cnt) {
  extern __shared__ double sm[];
  __shared__ int s_rot;
  __shared__ unsigned long long s_maxrel;
  __shared__ double s_norm[1024];   // c <= 1024
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  double* Mw = use_smem ? sm : gwork;
  double* Ww = Mw + (size_t)c * r;
  for (int i = tid; i < c * r; i += blockDim.x) Mw[i] = Min[(size_t)(i / r) * ld + (i % r)];
  for (int i = tid; i < c * c; i += blockDim.x) Ww[i] = (i / c == i % c) ? 1.0 : 0.0;
  if (tid == 0 && cnt) cnt[0]++;
  __syncthreads();
  const int ce = c + (c & 1);
  const double tol = 1e-15;
  // ||M||_F^2 (invariant under the rotations): rows below 1e-33 of it (norm < 3e-17 sigma_1, far under the rank
  // cut of reading S6) are left alone -- pairs of noise rows would otherwise keep rotating for all 60 sweeps.
  for (int p = warp; p < c; p += nwarp) {
    double a = 0;
    for (int i = lane; i < r; i += 32) { double u = Mw[(size_t)p * r + i]; a += u * u; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) s_norm[p] = a;
  }
  __syncthreads();
  double fro2 = 0.0;
  for (int p = 0; p < c; p++) fro2 += s_norm[p];
  const double sinv = fro2 > 0.0 ? 1.0 / fro2 : 0.0;
  __syncthreads();
  if (c > 1) {
    for (int sweep = 0; sweep < 60; sweep++) {
      if (tid == 0) { s_rot = 0; s_maxrel = 0ull; }
      __syncthreads();
      for (int step = 0; step < ce - 1; step++) {
        for (int pi = warp; pi < ce / 2; pi += nwarp) {
          int p, q;
          if (pi == 0) { p = ce - 1; q = step; }
          else {
            p = step + pi; if (p >= ce - 1) p -= ce - 1;
            q = step - pi; if (q < 0) q += ce - 1;
          }
          if (p >= c || q >= c) continue;
          if (p > q) { int t = p; p = q; q = t; }
          double* xp = Mw + (size_t)p * r;
          double* xq = Mw + (size_t)q * r;
          double a = 0, b = 0, g = 0;
          const double u0 = lane < r ? xp[lane] : 0.0, v0 = lane < r ? xq[lane] : 0.0;   // first 32 entries stay in registers
          a = u0 * u0; b = v0 * v0; g = u0 * v0;
          for (int i = lane + 32; i < r; i += 32) {
            double u = xp[i], v = xq[i];
            a += u * u; b += v * v; g += u * v;
          }
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_xor_sync(0xffffffffu, a, o);
            b += __shfl_xor_sync(0xffffffffu, b, o);
            g += __shfl_xor_sync(0xffffffffu, g, o);
          }
          // scaled by 1 / ||M||_F^2: a, b in (1e-33, 1], so neither the test nor q below can under- or overflow
          a *= sinv; b *= sinv; g *= sinv;
          if (fmin(a, b) > 1e-33 && g * g > tol * tol * a * b) {
            // tan of the rotation angle, t = 2 g sign(d) / (|d| + sqrt(d^2 + 4 g^2)), d = b - a, from approximate
            // reciprocal / reciprocal square root + two Newton steps each (full precision, no IEEE division)
            const double d = b - a, q2 = d * d + 4.0 * g * g;
            const double t = 2.0 * (d >= 0.0 ? g : -g) * rcp_fast(fabs(d) + q2 * rsqrt_fast(q2));
            const double cs = rsqrt_fast(1.0 + t * t), sn = cs * t;
            if (lane < r) {
              xp[lane] = cs * u0 - sn * v0;
              xq[lane] = sn * u0 + cs * v0;
            }
            for (int i = lane + 32; i < r; i += 32) {
              double u = xp[i], v = xq[i];
              xp[i] = cs * u - sn * v;
              xq[i] = sn * u + cs * v;
            }
            double* wp = Ww + (size_t)p * c;
            double* wq = Ww + (size_t)q * c;
            for (int i = lane; i < c; i += 32) {
              double u = wp[i], v = wq[i];
              wp[i] = cs * u - sn * v;
              wq[i] = sn * u + cs * v;
            }
            if (lane == 0) {
              s_rot = 1;
              // largest squared relative off-diagonal g^2 / (a b) rotated in this sweep (positive doubles order like integers)
              atomicMax(&s_maxrel, (unsigned long long)__double_as_longlong(g * g * rcp_fast(a * b)));
            }
          }
        }
        __syncthreads();
      }
      const int rot = s_rot;
      const double maxrel2 = __longlong_as_double((long long)s_maxrel);
      __syncthreads();
      if (tid == 0 && cnt) cnt[1]++;
      // quadratic convergence: once every rotation of a sweep had |g| / sqrt(a b) < 1e-10 the next sweep would find
      // nothing above 1e-15, so it is not run
      if (!rot || maxrel2 < 1e-20) break;
    }
  }
  // norms, ranks (descending, ties by index), sorted outputs
  for (int p = warp; p < c; p += nwarp) {
    double a = 0;
    for (int i = lane; i < r; i += 32) { double u = Mw[(size_t)p * r + i]; a += u * u; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) s_norm[p] = sqrt(a);
  }
  __syncthreads();
  for (int p = warp; p < c; p += nwarp) {
    double np = s_norm[p];
    int rank = 0;
    for (int q = lane; q < c; q += 32) {
      double nq = s_norm[q];
      rank += (nq > np || (nq == np && q < p)) ? 1 : 0;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) rank += __shfl_xor_sync(0xffffffffu, rank, o);
    for (int i = lane; i < r; i += 32) Mout[(size_t)rank * r + i] = Mw[(size_t)p * r + i];
    for (int i = lane; i < c; i += 32) Wt[(size_t)rank * c + i] = Ww[(size_t)p * c + i];
    if (lane == 0) sig[rank] = np;
  }
}

void jacobi_rows(tn_handle* h, const double* Min, int ld, int c, int r, double* Mout, double* Wt, double* sig) {
  if (c > 1024) tn_throw(TN_ERR_ARG, "jacobi_rows: c = %d > 1024", c);
  size_t need = ((size_t)c * r + (size_t)c * c) * sizeof(double);
  TN_SMEM_OPT_IN(h, k_jacobi_rows, 200 * 1024);
  if (need <= 200 * 1024) {
    const int jt = std::min(1024, std::max(128, 32 * ((c + 1) / 2)));   // one warp per pair: fewer warps, cheaper barriers
    k_jacobi_rows<<<1, jt, need, h->stream>>>(Min, ld, c, r, Mout, Wt, sig, nullptr, 1, h->d_cnt);
    TN_LAUNCH_CHECK(h);
  } else {
    double* work = h->dalloc<double>((size_t)c * r + (size_t)c * c);
    k_jacobi_rows<<<1, 1024, 0, h->stream>>>(Min, ld, c, r, Mout, Wt, sig, work, 0, h->d_cnt);
    TN_LAUNCH_CHECK(h);
    h->dfree(work);
  }
}

// T[i][j] = Wt[j][i] / sqrt(max(sig[j], floor*sig[0]))   (0 when sig[0] == 0 or sig[j] == 0)
__global__ void k_svqb_T(const double* Wt, const double* sig, int k, double* T) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= k * k) return;
  int i = t / k, j = t % k;
  double s0 = sig[0], sj = sig[j];
  double sc = (s0 > 0.0 && sj > 0.0) ? rsqrt(fmax(sj, 1e-13 * s0)) : 0.0;
  T[t] = Wt[(size_t)j * k + i] * sc;
}

void orth_columns_jacobi(tn_handle* h, double* Y, i64 m, int k, int passes) {
  if (m <= 0 || k <= 0) return;
  DBuf<double> G(h, (size_t)k * k), Go(h, (size_t)k * k), Wt(h, (size_t)k * k), T(h, (size_t)k * k), sig(h, k);
  DBuf<double> Y2(h, (size_t)m * k);
  for (int p = 0; p < passes; p++) {
    gemm_rm(h, true, false, k, k, (int)m, Y, k, Y, k, G.p, k);
    jacobi_rows(h, G.p, k, k, k, Go.p, Wt.p, sig.p);
    k_svqb_T<<<cdiv((i64)k * k, 256), 256, 0, h->stream>>>(Wt.p, sig.p, k, T.p);
    TN_LAUNCH_CHECK(h);
    gemm_rm(h, false, false, (int)m, k, k, Y, k, T.p, k, Y2.p, k);
    TN_CUDA(cudaMemcpyAsync(Y, Y2.p, sizeof(double) * m * k, cudaMemcpyDeviceToDevice, h->stream));
  }
}

// ============================================================================================
// projector / fold maps
// ============================================================================================
__device__ __forceinline__ int pdep8(int v, int mask) {
  int out = 0, bit = 0;
  for (int i = 0; i < 8; i++)
    if ((mask >> i) & 1) { out |= ((v >> bit) & 1) << i; bit++; }
  return out;
}

// Yk[o][(a,cl)][s] = sum_ch wC[cl][ch] * Y[o][Pl[a]*n_i + Pi[ch]][s]
// one thread per (o, a, s): the n_i inputs are read once into registers and all n_cl outputs written from them
// (W1[cl][i] = sum_{ch: Pi ch = i} wC[cl][ch] in shared memory); n_i, n_cl <= 16
__global__ void __launch_bounds__(256) k_map_L_med(CellDev c, const double* __restrict__ Y, double* __restrict__ Yk, int outer,
                                                   int s) {
  __shared__ double W1[256];
  for (int e = threadIdx.x; e < c.nCl * c.n_i; e += blockDim.x) {
    const int cl = e / c.n_i, i = e % c.n_i;
    double w = 0.0;
    for (int ch = 0; ch < c.nCh; ch++)
      if (c.Pi[ch] == i) w += c.wC[cl * c.nCh + ch];
    W1[e] = w;
  }
  __syncthreads();
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  i64 total = (i64)outer * c.nA * s;
  if (t >= total) return;
  int is = (int)(t % s);
  int a = (int)((t / s) % c.nA);
  int o = (int)(t / ((i64)s * c.nA));
  const double* base = Y + ((i64)o * (c.n_l * c.n_i) + (i64)c.Pl[a] * c.n_i) * s + is;
  double v[16];
#pragma unroll
  for (int i = 0; i < 16; i++) v[i] = i < c.n_i ? base[(i64)i * s] : 0.0;
  double* dst = Yk + ((i64)o * c.nK + (i64)a * c.nCl) * s + is;
  for (int cl = 0; cl < c.nCl; cl++) {
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < 16; i++) acc += (i < c.n_i ? W1[cl * c.n_i + i] : 0.0) * v[i];
    dst[(i64)cl * s] = acc;
  }
}
// Y[o][(l,i)][s] = sum_{a: Pl a = l} sum_cl sum_{ch: Pi ch = i} wC[cl][ch] Yk[o][(a,cl)][s]
// one thread per (o, l, s): every Yk entry is read once, the n_i outputs accumulate in registers
// (W2[i][cl] = sum_{ch: Pi ch = i} wC[cl][ch] in shared memory)
__global__ void __launch_bounds__(256) k_map_LT_med(CellDev c, const double* __restrict__ Yk, double* __restrict__ Y, int outer,
                                                    int s, int nbits, int half) {
  __shared__ double W2[256];
  const int fc_mask = (~c.m_din) & (c.nCh - 1), nfc = c.nCh / c.n_i;
  for (int e = threadIdx.x; e < c.n_i * c.nCl; e += blockDim.x) {
    const int i = e / c.nCl, cl = e % c.nCl;
    const int c0 = pdep8(i, c.m_din);
    double w = 0.0;
    for (int fc = 0; fc < nfc; fc++) w += c.wC[cl * c.nCh + (c0 | pdep8(fc, fc_mask))];
    W2[e] = w;
  }
  __syncthreads();
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  i64 total = (i64)outer * c.n_l * s;
  if (t >= total) return;
  int is = (int)(t % s);
  int l = (int)((t / s) % c.n_l);
  int o = (int)(t / ((i64)s * c.n_l));
  int fa_mask = (~c.m_left) & (c.nA - 1);
  int nfa = c.nA / c.n_l;
  int a0 = pdep8(l, c.m_left);
  double acc[16];
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i] = 0.0;
  for (int fa = 0; fa < nfa; fa++) {
    const int a = a0 | pdep8(fa, fa_mask);
    const double* src = Yk + ((i64)o * c.nK + (i64)a * c.nCl) * s + is;
    for (int cl = 0; cl < c.nCl; cl++) {
      const double v = src[(i64)cl * s];
#pragma unroll
      for (int i = 0; i < 16; i++) acc[i] += (i < c.n_i ? W2[i * c.nCl + cl] : 0.0) * v;
    }
  }
  double* dst = Y + ((i64)o * (c.n_l * c.n_i) + (i64)l * c.n_i) * s + is;
#pragma unroll
  for (int i = 0; i < 16; i++)
    if (i < c.n_i) dst[(i64)i * s] = acc[i];
}
// Yk[o][(a,cl)][s] = Y[o][Pr[a]*n_o + Po[cl]][s]
__global__ void k_map_R(CellDev c, const double* Y, double* Yk, int outer, int s) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  i64 total = (i64)outer * c.nK * s;
  if (t >= total) return;
  int is = (int)(t % s);
  int k = (int)((t / s) % c.nK);
  int o = (int)(t / ((i64)s * c.nK));
  int a = k / c.nCl, cl = k % c.nCl;
  Yk[t] = Y[((i64)o * (c.n_r * c.n_o) + (i64)c.Pr[a] * c.n_o + c.Po[cl]) * s + is];
}
// Y[o][(r,oo)][s] = sum_{a: Pr a = r} sum_{cl: Po cl = oo} Yk[o][(a,cl)][s]
__global__ void k_map_RT(CellDev c, const double* Yk, double* Y, int outer, int s) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  int wr = c.n_r * c.n_o;
  i64 total = (i64)outer * wr * s;
  if (t >= total) return;
  int is = (int)(t % s);
  int ro = (int)((t / s) % wr);
  int o = (int)(t / ((i64)s * wr));
  int r = ro / c.n_o, oo = ro % c.n_o;
  int fa_mask = (~c.m_right) & (c.nA - 1), fc_mask = (~c.m_dout) & (c.nCl - 1);
  int nfa = c.nA / c.n_r, nfc = c.nCl / c.n_o;
  int a0 = pdep8(r, c.m_right), c0 = pdep8(oo, c.m_dout);
  double acc = 0.0;
  for (int fa = 0; fa < nfa; fa++) {
    int a = a0 | pdep8(fa, fa_mask);
    for (int fc = 0; fc < nfc; fc++) {
      int cl = c0 | pdep8(fc, fc_mask);
      acc += Yk[((i64)o * c.nK + (i64)a * c.nCl + cl) * s + is];
    }
  }
  Y[t] = acc;
}

void map_L(tn_handle* h, const CellDev& c, bool fold, const double* Y, double* Yk, int outer, int s) {
  if (fold) {   // Yk[o][a][s] = sum_r BhS[r][a] Y[o][r][s]
    if (tsgemm_batched(h, true, c.bh_rows, s, c.nA, c.BhS, c.nA, Y, s, (i64)c.bh_rows * s, Yk, s, (i64)c.nA * s, outer)) return;
    GemmDesc g;
    g.M = c.nA; g.N = s; g.K = c.bh_rows; g.B1 = outer;
    g.A = c.BhS; g.a_i = 1; g.a_k = c.nA;
    g.B = Y; g.b_b1 = (i64)c.bh_rows * s; g.b_k = s; g.b_j = 1;
    g.C = Yk; g.c_b1 = (i64)c.nA * s; g.c_i = s; g.c_j = 1;
    g.nsplit = 1;
    gemm_general(h, g);
  } else {
    i64 total = (i64)outer * c.nA * s;
    k_map_L_med<<<cdiv(total, 256), 256, 0, h->stream>>>(c, Y, Yk, outer, s);
    TN_LAUNCH_CHECK(h);
  }
}
void map_LT(tn_handle* h, const CellDev& c, bool fold, const double* Yk, double* Y, int outer, int s) {
  if (fold) {   // Y[o][r][s] = sum_a BhS[r][a] Yk[o][a][s]
    if (tsgemm_batched(h, false, c.bh_rows, s, c.nA, c.BhS, c.nA, Yk, s, (i64)c.nA * s, Y, s, (i64)c.bh_rows * s, outer)) return;
    GemmDesc g;
    g.M = c.bh_rows; g.N = s; g.K = c.nA; g.B1 = outer;
    g.A = c.BhS; g.a_i = c.nA; g.a_k = 1;
    g.B = Yk; g.b_b1 = (i64)c.nA * s; g.b_k = s; g.b_j = 1;
    g.C = Y; g.c_b1 = (i64)c.bh_rows * s; g.c_i = s; g.c_j = 1;
    g.nsplit = 1;
    gemm_general(h, g);
  } else {
    i64 total = (i64)outer * c.n_l * s;
    k_map_LT_med<<<cdiv(total, 256), 256, 0, h->stream>>>(c, Yk, Y, outer, s, 0, 0);
    TN_LAUNCH_CHECK(h);
  }
}
void map_R(tn_handle* h, const CellDev& c, const double* Y, double* Yk, int outer, int s) {
  i64 total = (i64)outer * c.nK * s;
  k_map_R<<<cdiv(total, 256), 256, 0, h->stream>>>(c, Y, Yk, outer, s);
  TN_LAUNCH_CHECK(h);
}
void map_RT(tn_handle* h, const CellDev& c, const double* Yk, double* Y, int outer, int s) {
  i64 total = (i64)outer * c.n_r * c.n_o * s;
  k_map_RT<<<cdiv(total, 256), 256, 0, h->stream>>>(c, Yk, Y, outer, s);
  TN_LAUNCH_CHECK(h);
}

// ============================================================================================
// Theta-core (site):  batch = k;  rows i = (x, b);  cols = g;  inner = y
// ============================================================================================
struct LdThA {
  const double* A;
  const int* Pd;
  int nB, pd, dy;
  __device__ __forceinline__ double operator()(int, int i, int y) const {
    int x = i / nB, b = i % nB;
    return __ldg(A + ((i64)x * pd + Pd[b]) * dy + y);
  }
};
struct LdThE {
  const double* Ek;
  int nK, g;
  __device__ __forceinline__ double operator()(int k, int y, int j) const {
    return __ldg(Ek + ((i64)y * nK + k) * g + j);
  }
};
struct StTh {
  double* Tc;
  const double *wA, *X, *Yc;
  int nK, nB, nCl, tshift, g;
  __device__ __forceinline__ void operator()(int k, int, int i, int j, double v) const {
    int x = i / nB, b = i % nB;
    int a = k / nCl, cl = k % nCl;
    double w = wA[a] * X[(a >> tshift) * nB + b] * Yc[b * nCl + cl];
    Tc[(((i64)x * nK + k) * nB + b) * g + j] = v * w;
  }
};
template <int BN>
static void launch_theta(tn_handle* h, const CellDev& c, const double* A, int dx, int dy, const double* Ek, int g,
                         double* Tc) {
  LdThA a{A, c.Pd, c.nB, c.n_d, dy};
  LdThE b{Ek, c.nK, g};
  StTh e{Tc, c.wA, c.X, c.Yc, c.nK, c.nB, c.nCl, c.tshift, g};
  int M = dx * c.nB;
  dim3 grid((unsigned)c.nK, (unsigned)cdiv(M, 64), (unsigned)cdiv(g, BN));
  k_gemm<64, BN, 16, 4, 1, true, true, LdThA, LdThE, StTh><<<grid, 128, 0, h->stream>>>(M, g, dy, 1, a, b, e);
  TN_LAUNCH_CHECK(h);
}
// small-K route (bgemm.cuh): rows gathered through Pd by pointer, weight hoisted to one product per output row
struct ArTh {
  const double* A;
  const int* Pd;
  int nB, pd, dy;
  __device__ __forceinline__ const double* operator()(int, int i) const {
    return A + ((i64)(i / nB) * pd + Pd[i % nB]) * dy;
  }
};
struct BrTh {   // row y of B for batch k: Ek[(y, k)][0..g)
  const double* Ek;
  int nK, g;
  __device__ __forceinline__ const double* operator()(int k, int y) const { return Ek + ((i64)y * nK + k) * g; }
};
struct EpTh {
  double* Tc;
  const double *wA, *X, *Yc;
  int nK, nB, nCl, tshift, g;
  static constexpr bool kReduce = false;
  struct Row { double* p; double w; };
  __device__ __forceinline__ Row row(int k, int i) const {
    const int x = i / nB, b = i % nB, a = k / nCl, cl = k % nCl;
    return Row{Tc + (((i64)x * nK + k) * nB + b) * g, wA[a] * X[(a >> tshift) * nB + b] * Yc[b * nCl + cl]};
  }
  __device__ __forceinline__ void put(Row& r, int, int j, double v) const { r.p[j] = v * r.w; }
  __device__ __forceinline__ void put2(Row& r, int, int j, double v0, double v1) const {
    if (((g | j) & 1) == 0) *reinterpret_cast<double2*>(r.p + j) = make_double2(v0 * r.w, v1 * r.w);   // 16-byte store
    else { r.p[j] = v0 * r.w; r.p[j + 1] = v1 * r.w; }
  }
};
void theta_core(tn_handle* h, const CellDev& c, const double* A, int dx, int dy, const double* Ek, int g,
                double* Tc) {
  h->st.flop_theta_build += 2.0 * dx * c.nB * (double)c.nK * dy * g;
  {
    ArTh ar{A, c.Pd, c.nB, c.n_d, dy};
    LdThE be{Ek, c.nK, g};
    EpTh ep{Tc, c.wA, c.X, c.Yc, c.nK, c.nB, c.nCl, c.tshift, g};
    BrTh br{Ek, c.nK, g};
    if ((((uintptr_t)Ek) & 15) == 0 && launch_bgemm_pipe(h, c.nK, dx * c.nB, g, dy, ar, br, ep)) return;
    if (launch_bgemm<true>(h, c.nK, dx * c.nB, g, dy, ar, be, ep)) return;
  }
  if (g <= 16) launch_theta<16>(h, c, A, dx, dy, Ek, g, Tc);
  else if (g <= 32) launch_theta<32>(h, c, A, dx, dy, Ek, g, Tc);
  else if (g <= 48) launch_theta<48>(h, c, A, dx, dy, Ek, g, Tc);
  else launch_theta<64>(h, c, A, dx, dy, Ek, g, Tc);
}

// ============================================================================================
// mediating-tensor pieces
// ============================================================================================
// one thread per (al, r, o, g): the n_i inputs are read ONCE into registers and all n_q outputs written from them
// (n_i, n_q <= 16; Bd in shared memory) -- the first version re-read every input n_q times through L2
__global__ void __launch_bounds__(256) k_med_apply_bd(const double* __restrict__ T1, const double* __restrict__ Bd,
                                                      double* __restrict__ Theta, int al, int n_o, int n_r, int n_i, int n_q,
                                                      int g) {
  __shared__ double sBd[256];
  for (int e = threadIdx.x; e < n_q * n_i; e += blockDim.x) sBd[e] = Bd[e];
  __syncthreads();
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  i64 total = (i64)al * n_r * n_o * g;
  if (t >= total) return;
  int ig = (int)(t % g);
  i64 u = t / g;
  int o = (int)(u % n_o); u /= n_o;
  int r = (int)(u % n_r);
  int a = (int)(u / n_r);
  const double* src = T1 + ((((i64)a * n_o + o) * n_r + r) * n_i) * g + ig;
  double v[16];
#pragma unroll
  for (int i = 0; i < 16; i++) v[i] = i < n_i ? src[(i64)i * g] : 0.0;
  double* dst = Theta + ((((i64)a * n_r + r) * n_o + o) * n_q) * g + ig;
  for (int q = 0; q < n_q; q++) {
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < 16; i++) acc += (i < n_i ? sBd[q * n_i + i] : 0.0) * v[i];
    dst[(i64)q * g] = acc;
  }
}
void med_apply_bd(tn_handle* h, const double* T1, const double* Bd, double* Theta, int al, int n_o, int n_r,
                  int n_i, int n_q, int g) {
  if (n_i > 16 || n_q > 16) tn_throw(TN_ERR_ARG, "mediating position: diagonal leg of %d x %d states (at most 16 x 16)", n_q, n_i);
  i64 total = (i64)al * n_r * n_o * g;
  k_med_apply_bd<<<cdiv(total, 256), 256, 0, h->stream>>>(T1, Bd, Theta, al, n_o, n_r, n_i, n_q, g);
  TN_LAUNCH_CHECK(h);
}
__global__ void k_med_outer_bd(const double* TL, const double* Bd, double* Theta, i64 rows, int n_i, int n_q,
                               int g) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  i64 total = rows * n_i * n_q * g;
  if (t >= total) return;
  int ig = (int)(t % g);
  i64 u = t / g;
  int q = (int)(u % n_q); u /= n_q;
  int i = (int)(u % n_i);
  i64 row = u / n_i;
  Theta[t] = TL[row * g + ig] * Bd[q * n_i + i];
}
void med_outer_bd(tn_handle* h, const double* TL, const double* Bd, double* Theta, i64 rows, int n_i, int n_q,
                  int g) {
  i64 total = rows * n_i * n_q * g;
  k_med_outer_bd<<<cdiv(total, 256), 256, 0, h->stream>>>(TL, Bd, Theta, rows, n_i, n_q, g);
  TN_LAUNCH_CHECK(h);
}
