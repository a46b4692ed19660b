// Orthonormalisation of tall-skinny blocks (a3: QR canonicalisation, subspace-iteration bases).
//
// Y [m x k] (row-major, ld = k, k <= 96) is orthonormalised in place by up to `passes` rounds of
// pivot-floored Cholesky-QR:   G = Y^T Y,  G = L L^T,  Y <- Y L^-T.
// One launch per round does  [apply the previous round's T] -> [Gram of the result with DMMA] ->
// [last CTA: ordered reduction of the per-CTA partial Grams, test ||G - I||, Cholesky, triangular
// inverse], so a round costs one kernel instead of (split-K GEMM, reduce, Jacobi, scale, GEMM, copy).
// Pivots below ~1e-11 max_i G_ii are replaced by that floor (reading S6): a rank-deficient or
// exactly-zero direction is scaled by a bounded factor instead of breaking the factorisation, and the
// next round (conditioning improved by ~1e6.5) finishes the job; exactly-zero columns stay zero.
// Rounds stop early (device flag) once ||G - I||_max is at rounding level.
#include "kernels.cuh"
#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace {

constexpr int OR_ROWS = 64, OR_THREADS = 256;

constexpr int OR_GS = 12, OR_MAXG = 16;   // two-level ordered reduction: groups of OR_GS CTAs
struct OrthCtl { unsigned top; int done; int rounds; int pad; unsigned grp[OR_MAXG]; };

__device__ __forceinline__ double rsqrt_newton(double x) {   // MUFU seed + two Newton steps: full precision, no IEEE sqrt / div
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double hx = 0.5 * x;
  y = y * (1.5 - hx * y * y);
  return y * (1.5 - hx * y * y);
}
__device__ __forceinline__ double block_max256(double v, double* sh) {
  const int tid = threadIdx.x;
  __syncthreads();
  sh[tid] = v;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (tid < o) sh[tid] = fmax(sh[tid], sh[tid + o]);
    __syncthreads();
  }
  double r = sh[0];
  __syncthreads();
  return r;
}

// Last stage of a round, run by ONE CTA on the reduced Gram matrix in shared memory (sG [k x k], ld KP + 1):
// test ||G - I||, pivot-floored Cholesky, triangular inverse, T = L^-T to global memory (zero-padded KP x KP).
// Returns (to all threads) 1 when Y is already orthonormal to rounding (no T written), 2 when ||G - I|| <= 1e-4
// (applying this T gives an orthonormal block to rounding, u * cond(G): no further round is needed), else 0.
template <int KP>
__device__ int orth_factor(double* sG, double* sX, double* s_red, int k, double tol, double frel, double* Tout) {
  constexpr int LG = KP + 1;
  const int tid = threadIdx.x;
  double dev = 0.0, md = 0.0;
  for (int idx = tid; idx < k * k; idx += OR_THREADS) {
    int i = idx / k, j = idx % k;
    double v = sG[i * LG + j];
    dev = fmax(dev, fabs(v - (i == j ? 1.0 : 0.0)));
    if (i == j) md = fmax(md, v);
  }
  dev = block_max256(dev, s_red);
  md = block_max256(md, s_red);
  if (dev <= tol) return 1;
  const double floor_ = frel * md;
  // ---- Cholesky G = L L^T fused with the triangular inverse X = L^-1, two barriers per column.
  // Column j of L is G'_ij / L_jj below the diagonal; the diagonal entry of sG keeps the updated pivot G'_jj (so
  // no thread overwrites what another still reads and L_jj = sqrt(max(G'_jj, floor)) is recomputed where needed).
  // X is kept with UNSCALED rows: row j of L^-1 is sX[j][:] / L_jj.
  // A pivot at or below the floor (rounding noise of the Gram matrix, c * eps * md) is replaced by the floor and
  // its sub-column is dropped: noise directions are scaled up by a bounded factor and are NOT used to
  // "orthogonalise" later columns -- dividing noise by noise gives O(1) multipliers and an exponentially
  // ill-conditioned L.  The next round sees them at a resolvable size.
  for (int idx = tid; idx < k * k; idx += OR_THREADS) sX[(idx / k) * LG + idx % k] = (idx / k == idx % k) ? 1.0 : 0.0;
  // thread (ty, tx) = (tid / 32, tid % 32) walks rows ty, ty + 8, ... and columns tx, tx + 32, ...: no divisions
  const int tx = tid & 31, ty = tid >> 5;
  for (int j = 0; j < k; j++) {
    __syncthreads();                                   // updates of step j - 1 (and the X initialisation) are complete
    double d = sG[j * LG + j];
    const bool floored = !(d > floor_);
    if (floored) d = floor_;
    // 1 / L_jj; pivots below 1e-290 (only possible when the whole block is that small) take the exact route
    const double inv = d > 1e-290 ? rsqrt_newton(d) : (d > 0.0 ? 1.0 / sqrt(d) : 0.0);
    for (int i = j + 1 + tid; i < k; i += OR_THREADS) sG[i * LG + j] = floored ? 0.0 : sG[i * LG + j] * inv;
    __syncthreads();
    if (floored) continue;
    if constexpr (KP <= 48) {
      // all operands of this column's updates are read into registers first, then written: no load waits on a store
      constexpr int NR = KP / 8, NC = (KP + 31) / 32;
      double li[NR], lc[NC], xj[NC], gv[NR][NC], xv[NR][NC];
  #pragma unroll
      for (int a = 0; a < NR; a++) {
        const int i = j + 1 + ty + 8 * a;
        li[a] = i < k ? sG[i * LG + j] : 0.0;
      }
  #pragma unroll
      for (int b = 0; b < NC; b++) {
        const int c = j + 1 + tx + 32 * b, c2 = tx + 32 * b;
        lc[b] = c < k ? sG[c * LG + j] : 0.0;
        xj[b] = c2 <= j ? sX[j * LG + c2] * inv : 0.0;
      }
  #pragma unroll
      for (int a = 0; a < NR; a++)
  #pragma unroll
        for (int b = 0; b < NC; b++) {
          const int i = j + 1 + ty + 8 * a, c = j + 1 + tx + 32 * b, c2 = tx + 32 * b;
          gv[a][b] = (i < k && c <= i) ? sG[i * LG + c] : 0.0;
          xv[a][b] = (i < k && c2 <= j) ? sX[i * LG + c2] : 0.0;
        }
  #pragma unroll
      for (int a = 0; a < NR; a++)
  #pragma unroll
        for (int b = 0; b < NC; b++) {
          const int i = j + 1 + ty + 8 * a, c = j + 1 + tx + 32 * b, c2 = tx + 32 * b;
          if (i < k && c <= i) sG[i * LG + c] = gv[a][b] - li[a] * lc[b];       // trailing update of G
          if (i < k && c2 <= j) sX[i * LG + c2] = xv[a][b] - li[a] * xj[b];     // rank-1 update of L^-1
        }
    } else {   // larger blocks: the fully unrolled, predicated form above is issue-bound; walk the valid ranges only
      for (int i = j + 1 + ty; i < k; i += OR_THREADS / 32) {
        const double lij = sG[i * LG + j];
        for (int c = j + 1 + tx; c <= i; c += 32) sG[i * LG + c] -= lij * sG[c * LG + j];        // trailing update of G
        for (int c = tx; c <= j; c += 32) sX[i * LG + c] -= lij * (sX[j * LG + c] * inv);         // rank-1 update of L^-1
      }
    }
  }
  __syncthreads();
  // T = L^-T (upper triangular), zero-padded to KP x KP
  for (int idx = tid; idx < KP * KP; idx += OR_THREADS) {
    int c = idx / KP, j = idx % KP;
    double v = 0.0;
    if (c <= j && j < k) {
      double d = sG[j * LG + j];
      if (!(d > floor_)) d = floor_;
      v = d > 1e-290 ? sX[j * LG + c] * rsqrt_newton(d) : (d > 0.0 ? sX[j * LG + c] / sqrt(d) : 0.0);
    }
    Tout[idx] = v;
  }
  return dev <= 1e-4 ? 2 : 0;
}

template <int KT>
__global__ void __launch_bounds__(OR_THREADS) k_orth_pass(double* __restrict__ Y, i64 m, int k, const double* __restrict__ Tin,
                                                          double* __restrict__ Tout, double* __restrict__ part, OrthCtl* ctl,
                                                          int do_gram, double tol, double frel) {
  constexpr int KP = 8 * KT, LD = smem_ld(KP), NQ = (KT + 7) / 8;
  extern __shared__ double sm[];
  __shared__ double s_red[OR_THREADS];
  __shared__ int s_last;
  if (ctl->done) return;
  double* sT = sm;
  double* sIn = sT + KP * LD;
  double* sOut = sIn + OR_ROWS * LD;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (Tin)
    for (int idx = tid; idx < KP * KP; idx += OR_THREADS) sT[(idx / KP) * LD + idx % KP] = Tin[idx];
  double g[NQ][KT][2];
#pragma unroll
  for (int q = 0; q < NQ; q++)
#pragma unroll
    for (int j = 0; j < KT; j++) g[q][j][0] = g[q][j][1] = 0.0;

  const i64 ntile = (m + OR_ROWS - 1) / OR_ROWS;
  for (i64 tile = blockIdx.x; tile < ntile; tile += gridDim.x) {
    const i64 r0 = tile * OR_ROWS;
    __syncthreads();
    for (int idx = tid; idx < OR_ROWS * KP; idx += OR_THREADS) {
      int r = idx / KP, c = idx % KP;
      i64 gr = r0 + r;
      sIn[r * LD + c] = (gr < m && c < k) ? Y[gr * k + c] : 0.0;
    }
    __syncthreads();
    const double* src = sIn;
    if (Tin) {
      double o[KT][2];
#pragma unroll
      for (int j = 0; j < KT; j++) o[j][0] = o[j][1] = 0.0;
#pragma unroll 4
      for (int kk = 0; kk < KP; kk += 4) {
        double a = sIn[(8 * warp + (lane >> 2)) * LD + kk + (lane & 3)];
#pragma unroll
        for (int j = 0; j < KT; j++) dmma884(o[j][0], o[j][1], a, sT[(kk + (lane & 3)) * LD + 8 * j + (lane >> 2)]);
      }
#pragma unroll
      for (int j = 0; j < KT; j++) {
        int row = 8 * warp + (lane >> 2), col = 8 * j + 2 * (lane & 3);
        sOut[row * LD + col] = o[j][0];
        sOut[row * LD + col + 1] = o[j][1];
      }
      __syncthreads();
      for (int idx = tid; idx < OR_ROWS * KP; idx += OR_THREADS) {
        int r = idx / KP, c = idx % KP;
        i64 gr = r0 + r;
        if (gr < m && c < k) Y[gr * k + c] = sOut[r * LD + c];
      }
      src = sOut;
    }
    if (do_gram) {
#pragma unroll
      for (int q = 0; q < NQ; q++) {
        const int ti = warp + 8 * q;
        if (ti < KT) {
#pragma unroll 4
          for (int rr = 0; rr < OR_ROWS; rr += 4) {
            const double* row = src + (rr + (lane & 3)) * LD + (lane >> 2);
            double a = row[8 * ti];
#pragma unroll
            for (int j = 0; j < KT; j++) dmma884(g[q][j][0], g[q][j][1], a, row[8 * j]);
          }
        }
      }
    }
  }
  if (!do_gram) return;
  // ---- partial Gram -> workspace; the last CTA to arrive reduces in CTA order (deterministic)
  double* mine = part + (size_t)blockIdx.x * KP * KP;
#pragma unroll
  for (int q = 0; q < NQ; q++) {
    const int ti = warp + 8 * q;
    if (ti < KT) {
#pragma unroll
      for (int j = 0; j < KT; j++) {
        int row = 8 * ti + (lane >> 2), col = 8 * j + 2 * (lane & 3);
        mine[row * KP + col] = g[q][j][0];
        mine[row * KP + col + 1] = g[q][j][1];
      }
    }
  }
  const int nb = gridDim.x, ngrp = (nb + OR_GS - 1) / OR_GS, grp = blockIdx.x / OR_GS;
  const int g0 = grp * OR_GS, g1 = min(nb, g0 + OR_GS);
  double* gpart = part + (size_t)nb * KP * KP;
  __threadfence();
  __syncthreads();
  if (tid == 0) s_last = (atomicAdd(&ctl->grp[grp], 1u) == (unsigned)(g1 - g0 - 1)) ? 1 : 0;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  for (int idx = tid; idx < KP * KP; idx += OR_THREADS) {   // level 1: this group's CTAs, in CTA order
    double s = 0.0;
#pragma unroll 4
    for (int b = g0; b < g1; b++) s += __ldcg(part + (size_t)b * KP * KP + idx);
    gpart[(size_t)grp * KP * KP + idx] = s;
  }
  __threadfence();
  __syncthreads();
  if (tid == 0) s_last = (atomicAdd(&ctl->top, 1u) == (unsigned)(ngrp - 1)) ? 1 : 0;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  constexpr int LG = KP + 1;
  double* sG = sm;
  double* sX = sm + KP * LG;
  for (int idx = tid; idx < KP * KP; idx += OR_THREADS) {   // level 2: groups in order
    double s = 0.0;
#pragma unroll 4
    for (int b = 0; b < ngrp; b++) s += __ldcg(gpart + (size_t)b * KP * KP + idx);
    sG[(idx / KP) * LG + idx % KP] = s;
  }
  __syncthreads();
  const int verdict = orth_factor<KP>(sG, sX, s_red, k, tol, frel, Tout);
  if (tid == 0) { ctl->top = 0; ctl->rounds++; if (verdict == 1) ctl->done = 1; }
  if (tid < OR_MAXG) ctl->grp[tid] = 0;
}

// All rounds of one orthonormalisation in ONE cooperative launch (grid <= resident CTAs): the rounds are separated
// by grid-wide barriers instead of kernel boundaries, which removes ~5 launches and their gaps from every call.
// Same arithmetic as k_orth_pass; the Gram partials are added in a different (also fixed) association.
template <int KT>
__global__ void __launch_bounds__(OR_THREADS) k_orth_coop(double* __restrict__ Y, i64 m, int k, double* __restrict__ Tbuf,
                                                          double* __restrict__ part, OrthCtl* ctl, int passes, double tol,
                                                          double frel) {
  constexpr int KP = 8 * KT, LD = smem_ld(KP), NQ = (KT + 7) / 8, LG = KP + 1;
  extern __shared__ double sm[];
  __shared__ double s_red[OR_THREADS];
  cg::grid_group grid = cg::this_grid();
  double* sT = sm;
  double* sIn = sT + KP * LD;
  double* sOut = sIn + OR_ROWS * LD;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nb = gridDim.x, ngrp = (nb + OR_GS - 1) / OR_GS;
  double* gpart = part + (size_t)nb * KP * KP;
  const i64 ntile = (m + OR_ROWS - 1) / OR_ROWS;
  bool last = false;   // set when the previous round reported ||G - I|| <= 1e-4: apply its T and stop
  for (int p = 0; p <= passes; p++) {
    const bool has_T = p > 0, do_gram = p < passes && !last;
    const double* Tin = Tbuf + (size_t)((p - 1) & 1) * KP * KP;
    double* Tout = Tbuf + (size_t)(p & 1) * KP * KP;
    __syncthreads();
    if (has_T)
      for (int idx = tid; idx < KP * KP; idx += OR_THREADS) sT[(idx / KP) * LD + idx % KP] = __ldcg(Tin + idx);
    double g[NQ][KT][2];
#pragma unroll
    for (int q = 0; q < NQ; q++)
#pragma unroll
      for (int j = 0; j < KT; j++) g[q][j][0] = g[q][j][1] = 0.0;
    for (i64 tile = blockIdx.x; tile < ntile; tile += nb) {
      const i64 r0 = tile * OR_ROWS;
      __syncthreads();
      for (int idx = tid; idx < OR_ROWS * KP; idx += OR_THREADS) {
        int r = idx / KP, c = idx % KP;
        i64 gr = r0 + r;
        sIn[r * LD + c] = (gr < m && c < k) ? Y[gr * k + c] : 0.0;
      }
      __syncthreads();
      const double* src = sIn;
      if (has_T) {
        double o[KT][2];
#pragma unroll
        for (int j = 0; j < KT; j++) o[j][0] = o[j][1] = 0.0;
#pragma unroll 4
        for (int kk = 0; kk < KP; kk += 4) {
          double a = sIn[(8 * warp + (lane >> 2)) * LD + kk + (lane & 3)];
#pragma unroll
          for (int j = 0; j < KT; j++) dmma884(o[j][0], o[j][1], a, sT[(kk + (lane & 3)) * LD + 8 * j + (lane >> 2)]);
        }
#pragma unroll
        for (int j = 0; j < KT; j++) {
          int row = 8 * warp + (lane >> 2), col = 8 * j + 2 * (lane & 3);
          sOut[row * LD + col] = o[j][0];
          sOut[row * LD + col + 1] = o[j][1];
        }
        __syncthreads();
        for (int idx = tid; idx < OR_ROWS * KP; idx += OR_THREADS) {
          int r = idx / KP, c = idx % KP;
          i64 gr = r0 + r;
          if (gr < m && c < k) Y[gr * k + c] = sOut[r * LD + c];
        }
        src = sOut;
      }
      if (do_gram) {
#pragma unroll
        for (int q = 0; q < NQ; q++) {
          const int ti = warp + 8 * q;
          if (ti < KT) {
#pragma unroll 4
            for (int rr = 0; rr < OR_ROWS; rr += 4) {
              const double* row = src + (rr + (lane & 3)) * LD + (lane >> 2);
              double a = row[8 * ti];
#pragma unroll
              for (int j = 0; j < KT; j++) dmma884(g[q][j][0], g[q][j][1], a, row[8 * j]);
            }
          }
        }
      }
    }
    if (!do_gram) break;
    double* mine = part + (size_t)blockIdx.x * KP * KP;
#pragma unroll
    for (int q = 0; q < NQ; q++) {
      const int ti = warp + 8 * q;
      if (ti < KT) {
#pragma unroll
        for (int j = 0; j < KT; j++) {
          int row = 8 * ti + (lane >> 2), col = 8 * j + 2 * (lane & 3);
          mine[row * KP + col] = g[q][j][0];
          mine[row * KP + col + 1] = g[q][j][1];
        }
      }
    }
    grid.sync();
    {   // every CTA reduces its slice of the KP x KP entries over all partials: thread (e, q) adds partials
        // 8q .. 8q+7 (eight loads in flight), thread e then adds the group sums in order -- fixed association
      const int E = KP * KP, e0 = (int)((i64)E * blockIdx.x / nb), e1 = (int)((i64)E * (blockIdx.x + 1) / nb);
      const int EL = e1 - e0, nq = (nb + 7) / 8;
      double* s_ps = sm;                               // EL * nq <= KP * KP <= the dynamic shared memory of this kernel
      __syncthreads();
      for (int w = tid; w < EL * nq; w += OR_THREADS) {
        const int e = w % EL, q = w / EL;
        double v[8];
#pragma unroll
        for (int u = 0; u < 8; u++) v[u] = 8 * q + u < nb ? __ldcg(part + (size_t)(8 * q + u) * E + e0 + e) : 0.0;
        double ssum = 0.0;
#pragma unroll
        for (int u = 0; u < 8; u++) ssum += v[u];
        s_ps[q * EL + e] = ssum;
      }
      __syncthreads();
      for (int e = tid; e < EL; e += OR_THREADS) {
        double ssum = 0.0;
        for (int q = 0; q < nq; q++) ssum += s_ps[q * EL + e];
        gpart[e0 + e] = ssum;
      }
    }
    grid.sync();
    if (blockIdx.x == 0) {                 // factorisation of the reduced Gram matrix
      double* sG = sm;
      double* sX = sm + KP * LG;
      __syncthreads();
      for (int idx = tid; idx < KP * KP; idx += OR_THREADS) sG[(idx / KP) * LG + idx % KP] = __ldcg(gpart + idx);
      __syncthreads();
      const int verdict = orth_factor<KP>(sG, sX, s_red, k, tol, frel, Tout);
      if (tid == 0) { ctl->rounds++; if (verdict) ctl->done = verdict; }
    }
    grid.sync();
    const int verdict = *(volatile int*)&ctl->done;
    if (verdict == 1) break;
    last = verdict == 2;
  }
}

template <int KT>
void run_orth(tn_handle* h, double* Y, i64 m, int k, int passes) {
  constexpr int KP = 8 * KT, LD = smem_ld(KP);
  const size_t smem = sizeof(double) * ((size_t)KP * LD + 2 * (size_t)OR_ROWS * LD);
  TN_SMEM_OPT_IN(h, k_orth_pass<KT>, smem);
  int nb = (int)std::min<i64>(h->sms, (m + OR_ROWS - 1) / OR_ROWS);
  DBuf<double> part(h, (size_t)(nb + OR_MAXG) * KP * KP), T(h, 2 * (size_t)KP * KP);
  DBuf<OrthCtl> ctl(h, 1);
  TN_CUDA(cudaMemsetAsync(ctl.p, 0, sizeof(OrthCtl), h->stream));
  double tol = 1e-15 * (32.0 + std::sqrt((double)m));
  double frel = 1e-11 * std::max(1.0, std::sqrt((double)m) / 128.0);   // pivot floor relative to max_i G_ii
  // ---- one cooperative launch for all rounds when the device supports it and the grid is co-resident
  static int coop_slots_dev[64];
  static bool coop_known[64] = {false};
  const int dv = h->device & 63;
  if (!coop_known[dv]) {
    int coop = 0, occ = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, h->device);
    TN_CUDA(cudaFuncSetAttribute(k_orth_coop<KT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_orth_coop<KT>, OR_THREADS, smem);
    coop_slots_dev[dv] = coop ? h->sms * occ : 0;
    coop_known[dv] = true;
  }
  const int coop_slots = coop_slots_dev[dv];
  if (coop_slots > 0 && nb <= coop_slots) {
    double* Yp = Y;
    double* Tp = T.p;
    double* pp = part.p;
    OrthCtl* cp = ctl.p;
    void* args[] = {&Yp, &m, &k, &Tp, &pp, &cp, &passes, &tol, &frel};
    TN_CUDA(cudaLaunchCooperativeKernel((const void*)k_orth_coop<KT>, dim3(nb), dim3(OR_THREADS), args, smem, h->stream));
    TN_LAUNCH_CHECK(h);
    return;
  }
  for (int p = 0; p <= passes; p++) {
    const double* Tin = p > 0 ? T.p + (size_t)((p - 1) & 1) * KP * KP : nullptr;
    double* Tout = T.p + (size_t)(p & 1) * KP * KP;
    k_orth_pass<KT><<<nb, OR_THREADS, smem, h->stream>>>(Y, m, k, Tin, Tout, part.p, ctl.p, p < passes ? 1 : 0, tol, frel);
    TN_LAUNCH_CHECK(h);
  }
}

}  // namespace

void orth_columns_jacobi(tn_handle* h, double* Y, i64 m, int k, int passes);   // kernels.cu (k > 96)

void orth_columns(tn_handle* h, double* Y, i64 m, int k, int passes) {
  if (m <= 0 || k <= 0) return;
  h->st.flop_orth_svd += 2.0 * 4.0 * (double)m * k * k;
  if (k <= 16) run_orth<2>(h, Y, m, k, passes);
  else if (k <= 32) run_orth<4>(h, Y, m, k, passes);
  else if (k <= 48) run_orth<6>(h, Y, m, k, passes);
  else if (k <= 64) run_orth<8>(h, Y, m, k, passes);
  else if (k <= 80) run_orth<10>(h, Y, m, k, passes);
  else if (k <= 96) run_orth<12>(h, Y, m, k, passes);
  else orth_columns_jacobi(h, Y, m, k, passes);
}

// ---- tn_kernel_check: one building block on host data (kernel-level parity tests) ----------------
void kernel_check_run(tn_handle* h, int op, i64 m, int n, int k, const double* A, const double* B, double* C) {
  if (op == TN_CHECK_ORTH) {
    DBuf<double> Y(h, (size_t)m * k);
    TN_CUDA(cudaMemcpyAsync(Y.p, A, sizeof(double) * m * k, cudaMemcpyHostToDevice, h->stream));
    orth_columns(h, Y.p, m, k, 5);
    TN_CUDA(cudaMemcpyAsync(C, Y.p, sizeof(double) * m * k, cudaMemcpyDeviceToHost, h->stream));
    TN_CUDA(cudaStreamSynchronize(h->stream));
  } else if (op == TN_CHECK_GEMM_N || op == TN_CHECK_GEMM_T) {
    if (!B) tn_throw(TN_ERR_ARG, "B is NULL");
    const bool t = op == TN_CHECK_GEMM_T;
    const i64 nb = t ? m * n : (i64)k * n, nc = t ? (i64)k * n : m * n;
    DBuf<double> dA(h, (size_t)m * k), dB(h, (size_t)nb), dC(h, (size_t)nc);
    TN_CUDA(cudaMemcpyAsync(dA.p, A, sizeof(double) * m * k, cudaMemcpyHostToDevice, h->stream));
    TN_CUDA(cudaMemcpyAsync(dB.p, B, sizeof(double) * nb, cudaMemcpyHostToDevice, h->stream));
    if (t) gemm_rm(h, true, false, k, n, (int)m, dA.p, k, dB.p, n, dC.p, n);
    else gemm_rm(h, false, false, (int)m, n, k, dA.p, k, dB.p, n, dC.p, n);
    TN_CUDA(cudaMemcpyAsync(C, dC.p, sizeof(double) * nc, cudaMemcpyDeviceToHost, h->stream));
    TN_CUDA(cudaStreamSynchronize(h->stream));
  } else {
    tn_throw(TN_ERR_ARG, "unknown op %d", op);
  }
}

// ---- tn_kernel_bench: device time of one building block on device-resident random data -----------
void kernel_bench_run(tn_handle* h, int op, i64 m, int n, i64 k, int iters, double* ms_per_call) {
  if (iters < 1) iters = 1;
  cudaEvent_t e0, e1;
  TN_CUDA(cudaEventCreate(&e0)); TN_CUDA(cudaEventCreate(&e1));
  float ms = 0;
  if (op == TN_CHECK_ORTH) {
    DBuf<double> Y(h, (size_t)m * n), Y0(h, (size_t)m * n);
    fill_random(h, Y0.p, m * n, 7);
    double tot = 0;
    for (int it = -1; it < iters; it++) {
      TN_CUDA(cudaMemcpyAsync(Y.p, Y0.p, sizeof(double) * m * n, cudaMemcpyDeviceToDevice, h->stream));
      TN_CUDA(cudaEventRecord(e0, h->stream));
      orth_columns(h, Y.p, m, n, 5);
      TN_CUDA(cudaEventRecord(e1, h->stream));
      TN_CUDA(cudaEventSynchronize(e1));
      TN_CUDA(cudaEventElapsedTime(&ms, e0, e1));
      if (it >= 0) tot += ms;
    }
    *ms_per_call = tot / iters;
  } else if (op == TN_CHECK_GEMM_N || op == TN_CHECK_GEMM_T) {
    const bool t = op == TN_CHECK_GEMM_T;
    const i64 nb = t ? m * n : k * n, nc = t ? k * n : m * n;
    DBuf<double> dA(h, (size_t)m * k), dB(h, (size_t)nb), dC(h, (size_t)nc);
    fill_random(h, dA.p, m * k, 1);
    fill_random(h, dB.p, nb, 2);
    for (int it = -1; it < iters; it++) {
      if (it == 0) TN_CUDA(cudaEventRecord(e0, h->stream));
      if (t) gemm_rm(h, true, false, (int)k, n, (int)m, dA.p, (int)k, dB.p, n, dC.p, n);
      else gemm_rm(h, false, false, (int)m, n, (int)k, dA.p, (int)k, dB.p, n, dC.p, n);
    }
    TN_CUDA(cudaEventRecord(e1, h->stream));
    TN_CUDA(cudaEventSynchronize(e1));
    TN_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    *ms_per_call = ms / iters;
  } else {
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    tn_throw(TN_ERR_ARG, "unknown op %d", op);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
}
