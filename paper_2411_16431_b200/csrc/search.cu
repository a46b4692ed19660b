// a4(ii)-a5: branch and bound over cells.  Eq. (7) PAPER.md:94-98 (chain rule), Fig. 3
// (branch to d*M candidates, keep the M most probable), Eqs. (8)-(9) PAPER.md:100-107 (conditionals
// depend on the boundary only -> right blocks are computed once per row start and inherited),
// Fig. 6(b) PAPER.md:143 (fixed legs above, one open site, boundary MPS R_{y+1} below, contracted
// exactly, "up to normalization"), p_d PAPER.md:113.
//
// For beam element m at cell (x,y), with S, Q the tensors of R_{y+1} under columns x and x+1/2:
//   u(m;a,b,cl,ch) = hS[a] wA[a] X[t(a)][b] vS[b] Yc[b][cl] * (wC[cl][ch] dvec[Pi ch])
//                    * sum_{b''} LG_m[(Pd b, Po cl)][b''] RM_{m,x}[b''][Pr a],     LG_m = Lv_m . (S Q)
//   hS = BhS_x[Pr(a of the cell on the left)], vS = BvS_x[Pd(b of the cell above)], dvec = Bd_x[Po(c_lo of upper-left)].
#include "kernels.cuh"
#include "bgemm.cuh"
#include <algorithm>
#include <cfloat>
#include <map>
#include <memory>

namespace {

struct Cand { double score; int parent; unsigned state; };

struct RowTab {          // device tables of one column of the current row
  const CellDev* c;
  double* G = nullptr;   // [npp][Dl][Dr],  npp = n_d * n_o
  int Dl = 1, Dr = 1, npp = 1;
  double* RM = nullptr;  // [slot][Dr][n_r]
  double* ls = nullptr;  // [slot] log-scale of RM
};

// ---- functors ----------------------------------------------------------------------------------
struct LdLv { const double* Lv; int ld; __device__ __forceinline__ double operator()(int, int m, int k) const { return Lv[(i64)m * ld + k]; } };
struct LdGj { const double* G; int Dl, Dr; __device__ __forceinline__ double operator()(int, int k, int j) const { return __ldg(G + (i64)(j / Dr) * Dl * Dr + (i64)k * Dr + (j % Dr)); } };
struct StPlain { double* C; i64 ld; __device__ __forceinline__ void operator()(int, int, int i, int j, double v) const { C[(i64)i * ld + j] = v; } };

struct LdPA {   // A(m; i=(b,cl), k) = LG[m][(Pd b * n_o + Po cl)][k]
  const double* LG; const int *Pd, *Po; int nCl, n_o, npp, Dr;
  __device__ __forceinline__ double operator()(int m, int i, int k) const {
    int b = i / nCl, cl = i % nCl;
    return LG[((i64)m * npp + Pd[b] * n_o + Po[cl]) * Dr + k];
  }
};
struct LdPB {   // B(m; k, a) = RMc[m][k][a] = RM[slot m][k][Pr a] * hS[hrow m][a] * wA[a], materialised densely by k_rmc once per
                // cell: the column weights ride on the small operand (the epilogue of the conditional GEMM has only
                // row-wise factors left) and the B tile is read with coalesced loads instead of three dependent gathers
  const double* RMc; int Dr, nA;
  __device__ __forceinline__ double operator()(int m, int k, int a) const {
    return __ldg(RMc + ((i64)m * Dr + k) * nA + a);
  }
};
__global__ void k_rmc(const double* RM, const int* slot, const int* Pr, const double* hS, const double* wA, const int* hrow,
                      int nb, int Dr, int n_r, int nA, double* RMc) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (i64)nb * Dr * nA) return;
  const int a = (int)(t % nA), k = (int)((t / nA) % Dr), m = (int)(t / ((i64)nA * Dr));
  RMc[t] = RM[((i64)slot[m] * Dr + k) * n_r + Pr[a]] * (hS[(i64)hrow[m] * nA + a] * wA[a]);
}
struct StPV {
  double* V; const double *hS, *wA, *X, *vS, *Yc; const int *hrow, *vrow, *slot;
  int nA, nB, nCl, tshift; i64 per_m;
  __device__ __forceinline__ void operator()(int m, int, int i, int a, double acc) const {
    int b = i / nCl, cl = i % nCl;
    // (the column weights hS wA are already inside the B operand, LdPB)
    double w = X[(a >> tshift) * nB + b] * vS[(i64)vrow[slot[m]] * nB + b] * Yc[b * nCl + cl];
    V[(i64)m * per_m + (i64)i * nA + a] = acc * w;
  }
};
// small-K route (bgemm.cuh) for the conditionals: row pointer into LG, column weights cs[m][a] = hS wA precomputed
struct ArPV {
  const double* LG; const int *Pd, *Po; int nCl, n_o, npp, Dr;
  __device__ __forceinline__ const double* operator()(int m, int i) const {
    return LG + ((i64)m * npp + Pd[i / nCl] * n_o + Po[i % nCl]) * Dr;
  }
};
struct EpPV {   // stores V and, fused, collects Z_m = sum max(v, 0) fc[m][cl] and the count of negative entries
  double* V; const double *X, *vS, *Yc, *fc; const int *vrow, *slot;
  double* zpart; unsigned long long* nneg;
  int nA, nB, nCl, tshift, ntile; i64 per_m;
  static constexpr bool kReduce = true;
  struct Row { double* p; const double* x; double w, f, z; unsigned neg; };
  __device__ __forceinline__ Row row(int m, int i) const {
    const int b = i / nCl, cl = i % nCl;
    return Row{V + (i64)m * per_m + (i64)i * nA, X + b, vS[(i64)vrow[slot[m]] * nB + b] * Yc[b * nCl + cl],
               fc[(i64)m * nCl + cl], 0.0, 0u};
  }
  __device__ __forceinline__ void tally(Row& r, double v) const {   // the row factor fc[m][cl] is applied once, in collect
    r.z += fmax(v, 0.0);
    r.neg += v >= 0.0 ? 0u : 1u;   // negatives AND NaNs are counted (reading S7), as in the k_beam_Z route
  }
  __device__ __forceinline__ void put(Row& r, int, int a, double v) const {
    const double o = v * (r.w * r.x[(a >> tshift) * nB]);
    r.p[a] = o;
    tally(r, o);
  }
  __device__ __forceinline__ void put2(Row& r, int, int a, double v0, double v1) const {
    const double t0 = r.w * r.x[(a >> tshift) * nB];
    const double t1 = tshift > 0 && !(a & 1) ? t0 : r.w * r.x[((a + 1) >> tshift) * nB];   // a even: same a_hi
    const double o0 = v0 * t0, o1 = v1 * t1;
    if (((nA | a) & 1) == 0) *reinterpret_cast<double2*>(r.p + a) = make_double2(o0, o1);
    else { r.p[a] = o0; r.p[a + 1] = o1; }
    tally(r, o0);
    tally(r, o1);
  }
  __device__ __forceinline__ void collect(const Row& r, double& z, unsigned& n) const { z += r.z * r.f; n += r.neg; }
  __device__ __forceinline__ void tile_done(int m, int tile, double z, unsigned n) const {
    zpart[(i64)m * ntile + tile] = z;
    if (n) atomicAdd(nneg, (unsigned long long)n);
  }
};
// ---- conditionals, pipelined (round 2): V[m][(b,cl)][a] = w(b,cl) X[a_hi][b] sum_k LG[m][(Pd b, Po cl)][k] RMc[m][k][a]
// One CTA = (beam element m, 128 rows (b,cl)); its A tile (gathered rows of LG) stays in shared memory while the column
// tiles of the dense operand RMc[m] (32 columns each) stream through a cp.async double buffer, so loads of tile t+1,
// DMMAs of tile t and the weighted stores of tile t overlap; the X factors of a tile are requested before the multiply.
// Z_m = sum max(v, 0) fc[m][cl] and the count of negative / NaN entries come out of the epilogue as in EpPV.
struct CondArgs {
  const double* LG; const int *Pd, *Po; int nCl, n_o, npp, Dr;          // A rows
  const double* RMc; int nA;                                             // B: [m][Dr][nA]
  double* V; const double *X, *vS, *Yc, *fc; const int *vrow, *slot;     // epilogue
  double* zpart; unsigned long long* nneg;
  int nB, tshift, ntile, Mg; i64 per_m;
  double* rowmax;    // [m][Mg]: largest entry of every row of V (0 if none is positive); the selection reads it first
  int store;         // 0: V is NOT written (lazy mode: k_cond_rows writes the rows that reach the selection bound later)
  int tally;         // 0: Z partials and the negative count are not written (second run of the same cell)
};
template <int KP>
__global__ void __launch_bounds__(256, 3) k_cond(CondArgs a) {
  constexpr int BM = 128, NT = 4, BN = 8 * NT, LDA = smem_ld(KP), LDB = smem_ld(BN);
  extern __shared__ __align__(16) double cond_smem[];
  double* sA = cond_smem;
  double* sB = cond_smem + BM * LDA;            // two buffers of KP * LDB
  __shared__ double s_rz[8];
  __shared__ unsigned s_rn[8];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int m = blockIdx.x, m0 = blockIdx.y * BM, K = a.Dr, N = a.nA;
  const double* Bm = a.RMc + (i64)m * K * N;
  auto fetch = [&](int n0, int buf) {
    double* dst = sB + buf * (KP * LDB);
    constexpr int G = BN / 2;
    for (int idx = tid; idx < KP * G; idx += 256) {
      const int k = idx / G, g2 = 2 * (idx % G);
      const int rem = k < K ? N - (n0 + g2) : 0;
      const int bytes = rem >= 2 ? 16 : rem == 1 ? 8 : 0;
      const double* src = bytes ? Bm + (i64)k * N + n0 + g2 : Bm;
      unsigned sa = (unsigned)__cvta_generic_to_shared(dst + k * LDB + g2);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(src), "r"(bytes));
    }
    asm volatile("cp.async.commit_group;");
  };
  fetch(0, 0);
  for (int r = warp; r < BM; r += 8) {
    const int gi = m0 + r;
    const double* src = gi < a.Mg ? a.LG + ((i64)m * a.npp + a.Pd[gi / a.nCl] * a.n_o + a.Po[gi % a.nCl]) * K : nullptr;
#pragma unroll
    for (int k = lane; k < KP; k += 32) sA[r * LDA + k] = (src && k < K) ? __ldg(src + k) : 0.0;
  }
  // row descriptors of this thread's two rows
  const int row0 = m0 + 16 * warp + (lane >> 2), row1 = row0 + 8;
  const int sl = a.slot[m];
  double w[2], f[2], z[2] = {0.0, 0.0}, vmx[2] = {0.0, 0.0};
  const double* xr[2];
  double* vp[2];
  unsigned neg = 0;
#pragma unroll
  for (int i = 0; i < 2; i++) {
    const int row = i ? row1 : row0, rr = row < a.Mg ? row : 0, b = rr / a.nCl, cl = rr % a.nCl;
    w[i] = a.vS[(i64)a.vrow[sl] * a.nB + b] * a.Yc[b * a.nCl + cl];
    f[i] = a.fc[(i64)m * a.nCl + cl];
    xr[i] = a.X + b;
    vp[i] = a.V + (i64)m * a.per_m + (i64)rr * N;
  }
  const int ntn = (N + BN - 1) / BN;
  for (int t = 0; t < ntn; t++) {
    const int buf = t & 1, n0 = t * BN;
    if (t + 1 < ntn) {
      fetch(n0 + BN, buf ^ 1);
      asm volatile("cp.async.wait_group 1;");
    } else {
      asm volatile("cp.async.wait_group 0;");
    }
    __syncthreads();
    // X factors of this tile (columns a, a+1 share a_hi: tshift >= 1), requested before the multiply
    double xv[2][NT];
#pragma unroll
    for (int j = 0; j < NT; j++) {
      const int col = n0 + 8 * j + 2 * (lane & 3), cc = col < N ? col : 0;
      xv[0][j] = __ldg(xr[0] + (i64)(cc >> a.tshift) * a.nB);
      xv[1][j] = __ldg(xr[1] + (i64)(cc >> a.tshift) * a.nB);
    }
    const double* sb = sB + buf * (KP * LDB);
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
    __syncthreads();      // everyone is done with sb before the fetch of tile t + 2 overwrites it
#pragma unroll
    for (int i = 0; i < 2; i++) {
      if ((i ? row1 : row0) >= a.Mg) continue;
#pragma unroll
      for (int j = 0; j < NT; j++) {
        const int col = n0 + 8 * j + 2 * (lane & 3);
        if (col >= N) continue;
        const double s = w[i] * xv[i][j];
        const double o0 = acc[i][j][0] * s, o1 = acc[i][j][1] * s;
        if (a.store) *reinterpret_cast<double2*>(vp[i] + col) = make_double2(o0, o1);     // N even, col even
        z[i] += fmax(o0, 0.0) + fmax(o1, 0.0);
        vmx[i] = fmax(vmx[i], fmax(o0, o1));                                 // (fmax ignores NaNs)
        neg += (o0 >= 0.0 ? 0u : 1u) + (o1 >= 0.0 ? 0u : 1u);               // negatives and NaNs (reading S7)
      }
    }
  }
  if (a.rowmax) {   // the four lanes that share a row
#pragma unroll
    for (int i = 0; i < 2; i++) {
      double v = vmx[i];
      v = fmax(v, __shfl_xor_sync(0xffffffffu, v, 1));
      v = fmax(v, __shfl_xor_sync(0xffffffffu, v, 2));
      const int row = i ? row1 : row0;
      if ((lane & 3) == 0 && row < a.Mg) a.rowmax[(i64)m * a.Mg + row] = v;
    }
  }
  if (!a.tally) return;
  // ordered CTA reduction -> one partial per (m, row tile)
  double tz = z[0] * f[0] + z[1] * f[1];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    tz += __shfl_xor_sync(0xffffffffu, tz, o);
    neg += __shfl_xor_sync(0xffffffffu, neg, o);
  }
  if (lane == 0) { s_rz[warp] = tz; s_rn[warp] = neg; }
  __syncthreads();
  if (tid == 0) {
    double zz = 0.0;
    unsigned nn = 0;
    for (int q = 0; q < 8; q++) { zz += s_rz[q]; nn += s_rn[q]; }
    a.zpart[(i64)m * a.ntile + blockIdx.y] = zz;
    if (nn) atomicAdd(a.nneg, (unsigned long long)nn);
  }
}
template <int KP>
static void launch_cond_k(tn_handle* h, int nb, const CondArgs& a) {
  constexpr int LDA = smem_ld(KP), LDB = smem_ld(32);
  constexpr int smem = (int)sizeof(double) * (128 * LDA + 2 * KP * LDB);
  TN_SMEM_OPT_IN(h, k_cond<KP>, smem);
  k_cond<KP><<<dim3((unsigned)nb, (unsigned)a.ntile), 256, smem, h->stream>>>(a);
  TN_LAUNCH_CHECK(h);
}
// returns false when the shape does not fit (odd nA, X not shared by column pairs, bond > 64, too many row tiles)
static bool launch_cond(tn_handle* h, int nb, const CondArgs& a) {
  if (a.Dr < 1 || a.Dr > 64 || (a.nA & 1) || a.tshift < 1 || a.ntile > 65535 || (((uintptr_t)a.RMc) & 15) || (((uintptr_t)a.V) & 15))
    return false;
  if (a.Dr <= 16) launch_cond_k<16>(h, nb, a);
  else if (a.Dr <= 32) launch_cond_k<32>(h, nb, a);
  else if (a.Dr <= 48) launch_cond_k<48>(h, nb, a);
  else launch_cond_k<64>(h, nb, a);
  return true;
}

struct LdHA {   // A(i=(b',b''), kk=(b,cl)) = G[(Pd b * n_o + Po cl)][i]
  const double* G; const int *Pd, *Po; int nCl, n_o; i64 DD;
  __device__ __forceinline__ double operator()(int, int i, int kk) const {
    int b = kk / nCl, cl = kk % nCl;
    return __ldg(G + (i64)(Pd[b] * n_o + Po[cl]) * DD + i);
  }
};
struct LdHB {   // B(kk=(b,cl), j=(m,t)) = X[t][b] vS[vrow m][b] Yc[b][cl] fc[m][cl]
  const double *X, *vS, *Yc, *fc; const int* vrow; int nB, nCl, nT;
  __device__ __forceinline__ double operator()(int, int kk, int j) const {
    int b = kk / nCl, cl = kk % nCl, m = j / nT, t = j % nT;
    return X[t * nB + b] * vS[(i64)vrow[m] * nB + b] * Yc[b * nCl + cl] * fc[(i64)m * nCl + cl];
  }
};
// materialised operands of the right-block GEMM
__global__ void k_gather_G(const double* G, const int* Pd, const int* Po, int nCl, int n_o, i64 DD, int Kg, double* out) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (i64)Kg * DD) return;
  const int kk = (int)(t / DD);
  const i64 i = t % DD;
  out[t] = G[(i64)(Pd[kk / nCl] * n_o + Po[kk % nCl]) * DD + i];
}
__global__ void k_coef(const double* X, const double* vS, const double* Yc, const double* fc, const int* vrow, int nB, int nCl,
                       int nT, int Kg, int Ng, double* out) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (i64)Kg * Ng) return;
  const int kk = (int)(t / Ng), j = (int)(t % Ng);
  const int b = kk / nCl, cl = kk % nCl, m = j / nT, tt = j % nT;
  out[t] = X[tt * nB + b] * vS[(i64)vrow[m] * nB + b] * Yc[b * nCl + cl] * fc[(i64)m * nCl + cl];
}
// ---- right blocks, factorised (round 2).  coef_m[(b,cl); t] = X[t][b] vS_m[b] Yc[b][cl] fc_m[cl] is a product of a factor
// in (t, b) and a factor in (b, cl), so
//   H_m[i; t] = sum_b X[t][b] vS_m[b] ( sum_cl Gy[(b,cl)][i] fc_m[cl] ),   Gy[(b,cl)][i] = Yc[b][cl] G[(Pd b, Po cl)][i]
// costs 2 DD n_b (n_cl + n_T) FLOP per beam element instead of the 2 DD n_b n_cl n_T of the joint GEMM (8 x fewer for
// 16 x 16): plain FMA work on operands that stay in shared memory / L2, no intermediate in HBM.
// One CTA = 64 values of i = (b', b'') x 8 beam elements; thread = (i, 2 beam elements); b runs in chunks of 4 staged in
// shared memory.
__global__ void k_gather_Gy(const double* G, const double* Yc, const int* Pd, const int* Po, int nCl, int n_o, i64 DD, int Kg,
                            double* out) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (i64)Kg * DD) return;
  const int kk = (int)(t / DD);
  const i64 i = t % DD;
  out[t] = Yc[kk] * G[(i64)(Pd[kk / nCl] * n_o + Po[kk % nCl]) * DD + i];
}
// The same factorised contraction on the FP64 tensor cores (round 2, the default; the plain-FMA kernel below stays as
// TN_OPT_RBLOCK_FACT = 2 for the kernel-level comparison).  Per stage of BB = 4 values of b a CTA (64 values of i, 8 beam
// elements) runs two small DMMA products with the intermediate in shared memory; the G tile of the next stage arrives
// through a cp.async double buffer meanwhile:
//   phase 1  W_b[i][m] = sum_cl G[b][cl][i] fc[m][cl]          (A = G_b^T from shared memory, B = fc fragments in registers;
//            the per-beam factor vS_m[b] is applied to the accumulator fragment on its way to shared memory)
//   phase 2  H_m[i][t] += sum_b W[m][b][i] X[t][b]              (warp = beam element m; one k-step of 4 values of b per DMMA)
// Shared-memory strides are == 4 (mod 16) doubles between the four k rows of a fragment (conflict-free 8-byte reads).
template <int NTB>   // t blocks of 8: n_T <= 8 NTB
__global__ void __launch_bounds__(256, 2) k_rblock_mma(const double* __restrict__ Gy, const double* __restrict__ X,
                                                    const double* __restrict__ vS, const double* __restrict__ fc,
                                                    const int* __restrict__ vrow, int nb, int nB, int nCl, int nT, i64 DD,
                                                    double* __restrict__ H) {
  constexpr int BI = 64, BMM = 8, BB = 4, LDI = BI + 4, LDM = BB * LDI + 2, LDX = 8 * NTB + 4;
  extern __shared__ __align__(16) double rb_smem[];
  double* sG = rb_smem;                       // 2 x [BB][16][LDI]   G[b][cl][i], cp.async double buffer
  double* sW = sG + 2 * BB * 16 * LDI;        // [BMM][LDM]          W[m][b][i]  (row b at b * LDI)
  double* sX = sW + BMM * LDM;                // 2 x [BB][LDX]       X[t][b] of the stage
  double* sV = sX + 2 * BB * LDX;             // 2 x [BMM][BB]       vS[vrow m][b] of the stage
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, q = lane & 3;
  const i64 i0 = (i64)blockIdx.x * BI;
  const int m0 = blockIdx.y * BMM;
  const int ks = (nCl + 3) >> 2, ncl4 = 4 * ks;        // k-steps of phase 1 (rows cl >= nCl are zero-filled)
  // G tile of a stage: 16-byte cp.async (DD even, i0 a multiple of 64: a pair of i values is inside or outside together)
  auto fetch = [&](int b0, int buf) {
    double* dst = sG + buf * (BB * 16 * LDI);
    for (int e = tid; e < BB * ncl4 * (BI / 2); e += 256) {
      const int i2 = 2 * (e % (BI / 2)), cl = (e / (BI / 2)) % ncl4, bb = e / ((BI / 2) * ncl4);
      const bool in = cl < nCl && b0 + bb < nB && i0 + i2 < DD;
      const double* src = in ? Gy + ((i64)(b0 + bb) * nCl + cl) * DD + i0 + i2 : Gy;
      unsigned sa = (unsigned)__cvta_generic_to_shared(dst + (bb * 16 + cl) * LDI + i2);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(src), "r"(in ? 16 : 0));
    }
    asm volatile("cp.async.commit_group;");
  };
  fetch(0, 0);
  double ff[4];                                        // B fragments of phase 1: fc[m0 + g][4 s + q]
#pragma unroll
  for (int s4 = 0; s4 < 4; s4++) {
    const int cl = 4 * s4 + q, m = m0 + g;
    ff[s4] = (m < nb && cl < nCl) ? fc[(i64)m * nCl + cl] : 0.0;
  }
  double acc[8][NTB][2];
#pragma unroll
  for (int ib = 0; ib < 8; ib++)
#pragma unroll
    for (int tb = 0; tb < NTB; tb++) acc[ib][tb][0] = acc[ib][tb][1] = 0.0;
  int buf = 0;
  for (int b0 = 0; b0 < nB; b0 += BB, buf ^= 1) {
    // (sG[buf ^ 1] was last read in phase 1 of the previous stage, before that stage's second barrier)
    if (b0 + BB < nB) {
      fetch(b0 + BB, buf ^ 1);
      asm volatile("cp.async.wait_group 1;");
    } else {
      asm volatile("cp.async.wait_group 0;");
    }
    double* sXb = sX + buf * (BB * LDX);
    double* sVb = sV + buf * (BMM * BB);
    for (int e = tid; e < BB * 8 * NTB; e += 256) {
      const int t = e % (8 * NTB), bb = e / (8 * NTB);
      sXb[bb * LDX + t] = (t < nT && b0 + bb < nB) ? X[(i64)t * nB + b0 + bb] : 0.0;
    }
    if (tid < BMM * BB) {
      const int mm = tid / BB, bb = tid % BB, m = m0 + mm;
      sVb[mm * BB + bb] = (m < nb && b0 + bb < nB) ? vS[(i64)vrow[m] * nB + b0 + bb] : 0.0;
    }
    __syncthreads();
    const double* sGb = sG + buf * (BB * 16 * LDI);
    // phase 1: warp = block of 8 values of i, all BB values of b
#pragma unroll
    for (int bb = 0; bb < BB; bb++) {
      double c0 = 0.0, c1 = 0.0;
#pragma unroll
      for (int s4 = 0; s4 < 4; s4++)
        if (s4 < ks) dmma884(c0, c1, sGb[(bb * 16 + 4 * s4 + q) * LDI + warp * 8 + g], ff[s4]);
      // accumulator fragment: row i = 8 warp + g, columns m = 2 q, 2 q + 1
      sW[(2 * q) * LDM + bb * LDI + warp * 8 + g] = c0 * sVb[(2 * q) * BB + bb];
      sW[(2 * q + 1) * LDM + bb * LDI + warp * 8 + g] = c1 * sVb[(2 * q + 1) * BB + bb];
    }
    __syncthreads();
    // phase 2: warp = beam element, one k-step (the BB = 4 values of b)
    double fx[NTB];
#pragma unroll
    for (int tb = 0; tb < NTB; tb++) fx[tb] = sXb[q * LDX + tb * 8 + g];
#pragma unroll
    for (int ib = 0; ib < 8; ib++) {
      const double fa = sW[warp * LDM + q * LDI + ib * 8 + g];
#pragma unroll
      for (int tb = 0; tb < NTB; tb++) dmma884(acc[ib][tb][0], acc[ib][tb][1], fa, fx[tb]);
    }
  }
  const int m = m0 + warp;
  if (m >= nb) return;
#pragma unroll
  for (int ib = 0; ib < 8; ib++) {
    const i64 gi = i0 + ib * 8 + g;
    if (gi >= DD) continue;
#pragma unroll
    for (int tb = 0; tb < NTB; tb++)
#pragma unroll
      for (int e = 0; e < 2; e++) {
        const int t = tb * 8 + 2 * q + e;
        if (t < nT) H[((i64)m * nT + t) * DD + gi] = acc[ib][tb][e];
      }
  }
}
template <int NTB>
static void launch_rblock_mma(tn_handle* h, dim3 grid, const double* Gy, const double* X, const double* vS, const double* fc,
                              const int* vrow, int nb, int nB, int nCl, int nT, i64 DD, double* H) {
  constexpr int BI = 64, BMM = 8, BB = 4, LDI = BI + 4, LDM = BB * LDI + 2, LDX = 8 * NTB + 4;
  constexpr int smem = (int)sizeof(double) * (2 * BB * 16 * LDI + BMM * LDM + 2 * BB * LDX + 2 * BMM * BB);
  TN_SMEM_OPT_IN(h, k_rblock_mma<NTB>, smem);
  k_rblock_mma<NTB><<<grid, 256, smem, h->stream>>>(Gy, X, vS, fc, vrow, nb, nB, nCl, nT, DD, H);
  TN_LAUNCH_CHECK(h);
}
template <int NTT>   // NTT = number of a_hi values (n_T <= 16), compile-time bound of the accumulators
__global__ void __launch_bounds__(256, 2) k_rblock_h(const double* __restrict__ Gy, const double* __restrict__ X,
                                                  const double* __restrict__ vS, const double* __restrict__ fc,
                                                  const int* __restrict__ vrow, int nb, int nB, int nCl, int nT, i64 DD,
                                                  double* __restrict__ H) {
  constexpr int BI = 64, BMM = 8, BB = 4;           // i values, beam elements, b values per stage (32 KB of G per stage)
  __shared__ double sG[BB][16][BI];                 // [b][cl][i]
  __shared__ double sX[BB][NTT];                    // X[t][b] of the stage
  __shared__ double sF[BMM][16];                    // fc[m][cl]
  __shared__ double sV[BMM][BB];                    // vS[vrow m][b] of the stage
  const int tid = threadIdx.x, ti = tid & (BI - 1), tm = tid >> 6;        // 4 groups of 64 threads, 2 beam elements each
  const i64 i0 = (i64)blockIdx.x * BI;
  const int m0 = blockIdx.y * BMM;
  for (int e = tid; e < BMM * 16; e += 256) {
    const int mm = e / 16, cl = e % 16, m = m0 + mm;
    sF[mm][cl] = (m < nb && cl < nCl) ? fc[(i64)m * nCl + cl] : 0.0;
  }
  double acc[2][NTT];
#pragma unroll
  for (int q = 0; q < 2; q++)
#pragma unroll
    for (int t = 0; t < NTT; t++) acc[q][t] = 0.0;
  for (int b0 = 0; b0 < nB; b0 += BB) {
    __syncthreads();
    for (int e = tid; e < BB * nCl * BI; e += 256) {
      const int ii = e % BI, cl = (e / BI) % nCl, bb = e / (BI * nCl);
      const i64 gi = i0 + ii;
      sG[bb][cl][ii] = (b0 + bb < nB && gi < DD) ? Gy[((i64)(b0 + bb) * nCl + cl) * DD + gi] : 0.0;
    }
    for (int e = tid; e < BB * NTT; e += 256) {
      const int t = e % NTT, bb = e / NTT;
      sX[bb][t] = (t < nT && b0 + bb < nB) ? X[(i64)t * nB + b0 + bb] : 0.0;
    }
    if (tid < BMM * BB) {
      const int mm = tid / BB, bb = tid % BB, m = m0 + mm;
      sV[mm][bb] = (m < nb && b0 + bb < nB) ? vS[(i64)vrow[m] * nB + b0 + bb] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int bb = 0; bb < BB; bb++) {
      double w0 = 0.0, w1 = 0.0;
      for (int cl = 0; cl < nCl; cl++) {
        const double g = sG[bb][cl][ti];
        w0 += g * sF[2 * tm][cl];
        w1 += g * sF[2 * tm + 1][cl];
      }
      w0 *= sV[2 * tm][bb];
      w1 *= sV[2 * tm + 1][bb];
#pragma unroll
      for (int t = 0; t < NTT; t++) {
        const double xv = sX[bb][t];
        acc[0][t] += xv * w0;
        acc[1][t] += xv * w1;
      }
    }
  }
  const i64 gi = i0 + ti;
  if (gi < DD)
#pragma unroll
    for (int q = 0; q < 2; q++) {
      const int m = m0 + 2 * tm + q;
      if (m < nb)
#pragma unroll
        for (int t = 0; t < NTT; t++)
          if (t < nT) H[((i64)m * nT + t) * DD + gi] = acc[q][t];
    }
}

struct StH { double* H; i64 DD; __device__ __forceinline__ void operator()(int, int, int i, int j, double v) const { H[(i64)j * DD + i] = v; } };

// ---- small kernels -------------------------------------------------------------------------------
// vrow[x][m], drow[x][m] from the states of the row above
__global__ void k_above_rows(const unsigned* states, int ncell_ld, int nb, int y, int Lx, int ns, int S,
                             const CellDev* cells, int* vrow, int* drow) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nb * Lx) return;
  int x = t / nb, m = t % nb;
  int v = 0, d = 0;
  if (y > 0) {
    const int half = ns / 2;
    const CellDev& up = cells[(y - 1) * Lx + x];
    unsigned st = states[(i64)m * ncell_ld + (y - 1) * Lx + x];
    int b = S == 1 ? (st & ((1u << ns) - 1)) : ((st >> ns) & ((1u << ns) - 1));
    v = up.Pd[b];
    if (x > 0 && S == 3) {
      const CellDev& ul = cells[(y - 1) * Lx + x - 1];
      unsigned su = states[(i64)m * ncell_ld + (y - 1) * Lx + x - 1];
      d = ul.Po[(su >> (2 * ns)) & ((1u << half) - 1)];
    }
  }
  vrow[x * nb + m] = v;
  drow[x * nb + m] = d;
}
__global__ void k_hrow(const unsigned* states, int ncell_ld, int nb, int cellidx, int x, int ns, const CellDev* cells,
                       int* hrow) {
  int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= nb) return;
  int r = 0;
  if (x > 0) {
    unsigned st = states[(i64)m * ncell_ld + cellidx - 1];
    r = cells[cellidx - 1].Pr[st & ((1u << ns) - 1)];
  }
  hrow[m] = r;
}
// fc[m][cl] = sum_ch wC[cl][ch] Bd[drow][Pi ch]
__global__ void k_fc(CellDev c, const int* drow_x, const int* slot, int nb, double* fc) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nb * c.nCl) return;
  int m = t / c.nCl, cl = t % c.nCl;
  int dr = drow_x[slot ? slot[m] : m];
  double s = 0.0;
  for (int ch = 0; ch < c.nCh; ch++) s += c.wC[cl * c.nCh + ch] * c.Bd[dr * c.n_i + c.Pi[ch]];
  fc[t] = s;
}
// RS[m][b'][a] = wA[a] sum_b'' H[(m*nT + t(a))][b'][b''] RM[m][b''][Pr a]
__global__ void k_rs(CellDev c, const double* H, const double* RM, int nb, int Dl, int Dr, double* RS) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  i64 total = (i64)nb * Dl * c.nA;
  if (t >= total) return;
  int a = (int)(t % c.nA);
  int bl = (int)((t / c.nA) % Dl);
  int m = (int)(t / ((i64)c.nA * Dl));
  const double* hh = H + (((i64)m * c.nT + (a >> c.tshift)) * Dl + bl) * Dr;
  const double* rm = RM + (i64)m * Dr * c.n_r + c.Pr[a];
  double s = 0.0;
  for (int k = 0; k < Dr; k++) s += hh[k] * rm[(i64)k * c.n_r];
  RS[t] = c.wA[a] * s;
}
// per-m max-abs normalisation with log-scale
__global__ void k_norm_rm(double* RM, int per_m, const double* ls_in, double* ls_out) {
  __shared__ double sh[256];
  int m = blockIdx.x;
  double* p = RM + (i64)m * per_m;
  double mx = 0.0;
  for (int i = threadIdx.x; i < per_m; i += blockDim.x) mx = fmax(mx, fabs(p[i]));
  sh[threadIdx.x] = mx;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + o]);
    __syncthreads();
  }
  mx = sh[0];
  if (mx > 0.0)
    for (int i = threadIdx.x; i < per_m; i += blockDim.x) p[i] /= mx;
  if (threadIdx.x == 0) ls_out[m] = ls_in[m] + (mx > 0.0 ? log(mx) : 0.0);
}
// Z[m] = sum max(v,0) fc[m][cl]; negatives / NaNs counted and clamped in place (reading S7).  Grid (chunk, m):
// every CTA streams one contiguous chunk of V[m] with 16-byte loads; nA, nCl are powers of two (2^n_s, 2^(n_s/2)).
// Partial sums go to part[m][chunk]; k_beam_Z_final adds them in chunk order (deterministic).
__global__ void __launch_bounds__(256) k_beam_Z(double* V, i64 per_m, int lgA, int nCl, const double* fc, double* part,
                                                unsigned long long* nneg) {
  __shared__ double sh[256];
  __shared__ unsigned shn[256];
  const int m = blockIdx.y, nchunk = gridDim.x;
  const i64 per2 = per_m >> 1;                          // per_m is even (a power of two >= 4)
  const i64 c0 = per2 * blockIdx.x / nchunk, c1 = per2 * (blockIdx.x + 1) / nchunk;
  double2* v2 = reinterpret_cast<double2*>(V + (i64)m * per_m);
  const double* fcm = fc + (i64)m * nCl;
  double s = 0.0;
  unsigned neg = 0;
  for (i64 q = c0 + threadIdx.x; q < c1; q += 256) {
    double2 x = v2[q];
    const bool bad0 = !(x.x >= 0.0), bad1 = !(x.y >= 0.0);
    if (bad0 | bad1) {
      neg += (x.x < 0.0) + (x.y < 0.0);
      if (bad0) x.x = 0.0;
      if (bad1) x.y = 0.0;
      v2[q] = x;
    }
    const int cl = (int)(((2 * q) >> lgA) & (nCl - 1));   // both entries share (b, cl): nA is even
    s += (x.x + x.y) * fcm[cl];
  }
  sh[threadIdx.x] = s; shn[threadIdx.x] = neg;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) { sh[threadIdx.x] += sh[threadIdx.x + o]; shn[threadIdx.x] += shn[threadIdx.x + o]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) { part[(i64)m * nchunk + blockIdx.x] = sh[0]; if (shn[0]) atomicAdd(nneg, (unsigned long long)shn[0]); }
}
__global__ void k_beam_Z_final(const double* part, int nb, int nchunk, double* Z) {
  int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= nb) return;
  double s = 0.0;
  for (int c = 0; c < nchunk; c++) s += part[(i64)m * nchunk + c];
  Z[m] = s;
}
// scale[m] = exp(logp[m] - max logp) / Z[m]
__global__ void k_beam_scale(const double* logp, const double* Z, int nb, double* scale) {
  __shared__ double sh[256];
  double mx = -INFINITY;
  for (int i = threadIdx.x; i < nb; i += blockDim.x) mx = fmax(mx, logp[i]);
  sh[threadIdx.x] = mx;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + o]);
    __syncthreads();
  }
  mx = sh[0];
  // beam members more than 700 nats below the best keep a positive (clamped) scale: their children stay selectable when
  // fewer than M better candidates exist (the exact log-scores decide the final order, k_sel_score)
  for (int i = threadIdx.x; i < nb; i += blockDim.x) scale[i] = Z[i] > 0.0 ? exp(fmax(logp[i] - mx, -700.0)) / Z[i] : 0.0;
  if (threadIdx.x == 0) scale[nb] = mx;   // key r = v fcd scale_m  <=>  score = log r + mx
}

// ---- top-M radix selection on r = v * fcd * scale (monotone in the score) ------------------------
struct SelState {
  unsigned long long prefix;   // key bits fixed so far (above `shift`)
  unsigned long long want;     // rank still to locate inside the prefix class
  unsigned long long above;    // candidates strictly above the prefix class
  unsigned long long inbin;    // candidates inside the prefix class
  unsigned long long thresh;   // final threshold key
  int done, takeall;
};
struct SelArgs {
  const double* V; const double *scale, *wC, *Bd; const int *drow_x, *slot, *Pi;
  i64 per_m; int nb, nA, nCl, nCh, n_i;
};
__device__ __forceinline__ double sel_fcd(const SelArgs& a, int m, int cl, int ch) {
  return a.wC[cl * a.nCh + ch] * a.Bd[a.drow_x[a.slot[m]] * a.n_i + a.Pi[ch]];
}
__device__ __forceinline__ unsigned long long sel_mix(unsigned long long z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
// Histogram of one radix digit of the keys.  sample_log2 > 0: only one hashed element of every
// 2^sample_log2 consecutive entries of V is looked at (a SUBSET of the candidates: its (M+1)-th largest key is a
// guaranteed lower bound of the true (M+1)-th largest, used as a prefilter threshold).
__global__ void k_sel_hist(SelArgs a, const SelState* st, int shift, int nbits, int first, int sample_log2, unsigned* hist) {
  __shared__ unsigned sh[4096];
  for (int i = threadIdx.x; i < 4096; i += blockDim.x) sh[i] = 0;
  __syncthreads();
  const unsigned long long prefix = st->prefix;
  const i64 total = (i64)a.nb * a.per_m;
  const i64 nq = sample_log2 ? ((total + (1ll << sample_log2) - 1) >> sample_log2) : total;
  for (i64 q = (i64)blockIdx.x * blockDim.x + threadIdx.x; q < nq; q += (i64)gridDim.x * blockDim.x) {
    i64 t = q;
    if (sample_log2) {
      t = (q << sample_log2) + (i64)(sel_mix((unsigned long long)q) & ((1ull << sample_log2) - 1));
      if (t >= total) continue;
    }
    double v = a.V[t];
    if (!(v > 0.0)) continue;
    int m = (int)(t / a.per_m);
    int cl = (int)(((t % a.per_m) / a.nA) % a.nCl);
    double vs = v * a.scale[m];
    for (int ch = 0; ch < a.nCh; ch++) {
      double r = vs * sel_fcd(a, m, cl, ch);
      if (!(r > 0.0)) continue;
      unsigned long long key = (unsigned long long)__double_as_longlong(r);
      if (!first && (key >> (shift + nbits)) != prefix) continue;
      atomicAdd(&sh[(key >> shift) & ((1u << nbits) - 1)], 1u);
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 4096; i += blockDim.x)
    if (sh[i]) atomicAdd(&hist[i], sh[i]);
}
// Locates the bin (scanning from the top) that holds the `want`-th largest key.  One CTA of 1024 threads,
// 4 bins per thread in descending order, block-wide inclusive scan.
__global__ void __launch_bounds__(1024) k_sel_resolve(SelState* st, unsigned* hist, int shift, int nbits, int first,
                                                      unsigned long long cap) {
  __shared__ unsigned long long sc[1024];
  __shared__ int s_found;
  __shared__ unsigned long long s_cum, s_inbin;
  const int tid = threadIdx.x, nbin = 1 << nbits;
  if (tid == 0) s_found = -1;
  unsigned hb[4];
  unsigned long long sum = 0;
#pragma unroll
  for (int j = 0; j < 4; j++) {
    int b = nbin - 1 - (4 * tid + j);
    hb[j] = b >= 0 ? hist[b] : 0u;
    sum += hb[j];
  }
  sc[tid] = sum;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    unsigned long long v = tid >= o ? sc[tid - o] : 0ull;
    __syncthreads();
    sc[tid] += v;
    __syncthreads();
  }
  const unsigned long long want = st->want;
  unsigned long long cum = sc[tid] - sum;
#pragma unroll
  for (int j = 0; j < 4; j++) {
    int b = nbin - 1 - (4 * tid + j);
    if (b >= 0 && cum < want && cum + hb[j] >= want) { s_found = b; s_cum = cum; s_inbin = hb[j]; }
    cum += hb[j];
  }
  const unsigned long long totalc = sc[1023];
  __syncthreads();
  for (int b = tid; b < 4096; b += 1024) hist[b] = 0;
  if (tid) return;
  const int found = s_found;
  if (found < 0) {            // fewer candidates than wanted: take everything positive
    st->takeall = 1; st->done = 1; st->thresh = 1ull;
    st->inbin = 0; st->above += totalc;
  } else {
    st->prefix = first ? (unsigned long long)found : ((st->prefix << nbits) | (unsigned long long)found);
    st->want -= s_cum;
    st->above += s_cum;
    st->inbin = s_inbin;
    st->thresh = st->prefix << shift;
    if (st->above + st->inbin <= cap || shift == 0) st->done = 1;
  }
}
struct Raw { int m; int i; int a; int ch; };
__global__ void k_sel_collect(SelArgs a, const SelState* st, Raw* out, unsigned* count, unsigned cap) {
  double thr = __longlong_as_double((long long)st->thresh);
  thr = st->takeall ? 0.0 : thr * (1.0 - 1e-12);
  const i64 total = (i64)a.nb * a.per_m;
  for (i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (i64)gridDim.x * blockDim.x) {
    double v = a.V[t];
    if (!(v > 0.0)) continue;
    int m = (int)(t / a.per_m);
    i64 rem = t % a.per_m;
    int i = (int)(rem / a.nA), aa = (int)(rem % a.nA);
    int cl = i % a.nCl;
    double vs = v * a.scale[m];
    for (int ch = 0; ch < a.nCh; ch++) {
      double r = vs * sel_fcd(a, m, cl, ch);
      if (r > 0.0 && r >= thr) {
        unsigned idx = atomicAdd(count, 1u);
        if (idx < cap) out[idx] = Raw{m, i, aa, ch};
      }
    }
  }
}
// Histogram of one radix digit of the keys of the ROW MAXIMA (one candidate per row (m, b, c_lo): the row's largest entry
// with its best c_hi).  A subset of the candidates, so its (M+1)-th largest key is a lower bound of the true (M+1)-th
// largest -- the prefilter threshold -- from 8 bytes per row (written by k_cond) instead of a scattered sample of V.
__global__ void k_sel_hist_rows(const double* rowmax, const double* scale, const double* fmx, int nb, int Mg, int nCl,
                                const SelState* st, int shift, int nbits, int first, unsigned* hist) {
  __shared__ unsigned sh[4096];
  for (int i = threadIdx.x; i < 4096; i += blockDim.x) sh[i] = 0;
  __syncthreads();
  const unsigned long long prefix = st->prefix;
  const i64 total = (i64)nb * Mg;
  for (i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (i64)gridDim.x * blockDim.x) {
    const int m = (int)(t / Mg), cl = (int)(t % Mg) % nCl;
    const double r = rowmax[t] * scale[m] * fmx[(i64)m * nCl + cl];
    if (!(r > 0.0)) continue;
    const unsigned long long key = (unsigned long long)__double_as_longlong(r);
    if (!first && (key >> (shift + nbits)) != prefix) continue;
    atomicAdd(&sh[(key >> shift) & ((1u << nbits) - 1)], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 4096; i += blockDim.x)
    if (sh[i]) atomicAdd(&hist[i], sh[i]);
}
// fmx[m][cl] = max_ch fcd(m, cl, ch): upper bound used to reject whole (m,i,a) entries with one compare
__global__ void k_sel_fmax(SelArgs a, double* fmx, int* chbest = nullptr) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= a.nb * a.nCl) return;
  int m = t / a.nCl, cl = t % a.nCl;
  double mx = 0.0;
  int best = 0;
  for (int ch = 0; ch < a.nCh; ch++) {
    const double f = sel_fcd(a, m, cl, ch);
    if (f > mx) { mx = f; best = ch; }     // the lowest c_hi among equal maxima (S8 order)
  }
  fmx[t] = mx;
  if (chbest) chbest[t] = best;
}
// ---- lazy V (round 2, TN_OPT_LAZY_V): k_cond ran with store = 0 (row maxima, Z and the negative count only: no 8 B per
// entry to HBM); once the selection bound is known, this kernel recomputes the rows whose maximum reaches it and writes
// them to their places in V, where the prefilter (same row test) and k_sel_score read them.  Same DMMA sequence per
// entry as k_cond (k ascending in steps of 4 from a zero accumulator, then one multiply by the same weight), so the
// recomputed entries equal the ones the row maxima came from.  Grid (row chunks of 1024, m); a warp takes 8 listed rows.
template <int KP>
__global__ void __launch_bounds__(256) k_cond_rows(CondArgs a, const SelState* st, const double* scale, const double* fmx) {
  constexpr int NT = 4, BN = 8 * NT;
  __shared__ int s_list[1024];
  __shared__ int s_cnt;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int m = blockIdx.y, r0 = blockIdx.x * 1024, K = a.Dr, N = a.nA;
  if (tid == 0) s_cnt = 0;
  __syncthreads();
  double thr = __longlong_as_double((long long)st->thresh);
  thr = st->takeall ? 0.0 : thr * (1.0 - 1e-12);
  const double sc = scale[m];
  for (int r = r0 + tid; r < min(r0 + 1024, a.Mg); r += 256) {
    const int cl = r % a.nCl;
    if (a.rowmax[(i64)m * a.Mg + r] * sc * fmx[(i64)m * a.nCl + cl] >= thr) s_list[atomicAdd(&s_cnt, 1)] = r;   // the prefilter's test
  }
  __syncthreads();
  const int cnt = s_cnt;
  const double* Bm = a.RMc + (i64)m * K * N;
  const int sl = a.slot[m];
  for (int g = warp; g * 8 < cnt; g += 8) {
    const int li = g * 8 + (lane >> 2);
    const bool live = li < cnt;
    const int row = live ? s_list[li] : 0, b = row / a.nCl, cl = row % a.nCl;
    const double* src = a.LG + ((i64)m * a.npp + a.Pd[b] * a.n_o + a.Po[cl]) * K;
    double fa[KP / 4];
#pragma unroll
    for (int q = 0; q < KP / 4; q++) {
      const int k = 4 * q + (lane & 3);
      fa[q] = (live && k < K) ? __ldg(src + k) : 0.0;
    }
    const double w = a.vS[(i64)a.vrow[sl] * a.nB + b] * a.Yc[b * a.nCl + cl];
    const double* xr = a.X + b;
    double* vp = a.V + (i64)m * a.per_m + (i64)row * N;
    for (int n0 = 0; n0 < N; n0 += BN) {
      double acc[NT][2];
#pragma unroll
      for (int j = 0; j < NT; j++) acc[j][0] = acc[j][1] = 0.0;
#pragma unroll
      for (int q = 0; q < KP / 4; q++) {
        const int k = 4 * q + (lane & 3);
#pragma unroll
        for (int j = 0; j < NT; j++) {
          const int col = n0 + 8 * j + (lane >> 2);
          const double fb = (k < K && col < N) ? __ldg(Bm + (i64)k * N + col) : 0.0;
          dmma884(acc[j][0], acc[j][1], fa[q], fb);
        }
      }
      if (!live) continue;
#pragma unroll
      for (int j = 0; j < NT; j++) {
        const int col = n0 + 8 * j + 2 * (lane & 3);
        if (col >= N) continue;
        const double s = w * __ldg(xr + (i64)(col >> a.tshift) * a.nB);
        *reinterpret_cast<double2*>(vp + col) = make_double2(acc[j][0] * s, acc[j][1] * s);
      }
    }
  }
}
static void launch_cond_rows(tn_handle* h, int nb, const CondArgs& a, const SelState* st, const double* scale, const double* fmx) {
  const dim3 grid((unsigned)((a.Mg + 1023) / 1024), (unsigned)nb);
  if (a.Dr <= 16) k_cond_rows<16><<<grid, 256, 0, h->stream>>>(a, st, scale, fmx);
  else if (a.Dr <= 32) k_cond_rows<32><<<grid, 256, 0, h->stream>>>(a, st, scale, fmx);
  else if (a.Dr <= 48) k_cond_rows<48><<<grid, 256, 0, h->stream>>>(a, st, scale, fmx);
  else k_cond_rows<64><<<grid, 256, 0, h->stream>>>(a, st, scale, fmx);
  TN_LAUNCH_CHECK(h);
}
// Prefilter pass over all of V: candidates with key >= thr go to the compact list (keys + Raw).  Grid (chunk, m),
// 16-byte loads, shifts instead of divisions (nA, nCl powers of two); survivors are rare.
__global__ void __launch_bounds__(256) k_sel_prefilter(SelArgs a, int lgA, const SelState* st, const double* fmx, double* keys,
                                                       Raw* out, unsigned* count, unsigned cap, const double* rowmax = nullptr) {
  double thr = __longlong_as_double((long long)st->thresh);
  thr = st->takeall ? 0.0 : thr * (1.0 - 1e-12);
  const int m = blockIdx.y, nchunk = gridDim.x;
  const i64 per2 = a.per_m >> 1;
  const i64 c0 = per2 * blockIdx.x / nchunk, c1 = per2 * (blockIdx.x + 1) / nchunk;
  const double2* v2 = reinterpret_cast<const double2*>(a.V + (i64)m * a.per_m);
  const double sc = a.scale[m];
  const double* fm = fmx + (i64)m * a.nCl;
  if (rowmax) {
    // one test per ROW (a lane per row, 32 rows per warp step); the warp then walks the rows that passed together, so
    // the cost is the 8 B per row of the maxima plus the few rows that reach the bound
    const double* rmx = rowmax + (i64)m * (a.per_m >> lgA);
    const int nrows = (int)(a.per_m >> lgA), rpc = (nrows + nchunk - 1) / nchunk;
    const int r0 = blockIdx.x * rpc, r1 = min(nrows, r0 + rpc);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, half = a.nA >> 1;
    for (int base = r0 + 32 * warp; base < r1; base += 256) {
      const int ri = base + lane;
      unsigned mask = __ballot_sync(0xffffffffu, ri < r1 && rmx[ri] * sc * fm[ri & (a.nCl - 1)] >= thr);
      while (mask) {
        const int i = base + __ffs(mask) - 1, cl = i & (a.nCl - 1);
        mask &= mask - 1;
        for (int qq = lane; qq < half; qq += 32) {
          const double2 x = v2[(i64)i * half + qq];
          const double bound = fmax(x.x, x.y) * sc * fm[cl];
          if (!(bound >= thr) || !(bound > 0.0)) continue;
#pragma unroll
          for (int e = 0; e < 2; e++) {
            const double v = e ? x.y : x.x;
            if (!(v > 0.0)) continue;
            const double vs = v * sc;
            const int aa = 2 * qq + e;
            for (int ch = 0; ch < a.nCh; ch++) {
              double r = vs * sel_fcd(a, m, cl, ch);
              if (r > 0.0 && r >= thr) {
                unsigned idx = atomicAdd(count, 1u);
                if (idx < cap) { keys[idx] = r; out[idx] = Raw{m, i, aa, ch}; }
              }
            }
          }
        }
      }
    }
    return;
  }
  for (i64 q = c0 + threadIdx.x; q < c1; q += 256) {
    const int i = (int)((2 * q) >> lgA), cl = i & (a.nCl - 1);
    const double2 x = v2[q];
    const double bound = fmax(x.x, x.y) * sc * fm[cl];
    if (!(bound >= thr) || !(bound > 0.0)) continue;
#pragma unroll
    for (int e = 0; e < 2; e++) {
      const double v = e ? x.y : x.x;
      if (!(v > 0.0)) continue;
      const double vs = v * sc;
      const int aa = (int)((2 * q + e) & (a.nA - 1));
      for (int ch = 0; ch < a.nCh; ch++) {
        double r = vs * sel_fcd(a, m, cl, ch);
        if (r > 0.0 && r >= thr) {
          unsigned idx = atomicAdd(count, 1u);
          if (idx < cap) { keys[idx] = r; out[idx] = Raw{m, i, aa, ch}; }
        }
      }
    }
  }
}
// radix digit histogram / final compaction on the compact key list
__global__ void k_csel_hist(const double* keys, unsigned n, const SelState* st, int shift, int nbits, int first, unsigned* hist) {
  __shared__ unsigned sh[4096];
  for (int i = threadIdx.x; i < 4096; i += blockDim.x) sh[i] = 0;
  __syncthreads();
  const unsigned long long prefix = st->prefix;
  for (unsigned t = blockIdx.x * blockDim.x + threadIdx.x; t < n; t += gridDim.x * blockDim.x) {
    unsigned long long key = (unsigned long long)__double_as_longlong(keys[t]);
    if (!first && (key >> (shift + nbits)) != prefix) continue;
    atomicAdd(&sh[(key >> shift) & ((1u << nbits) - 1)], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 4096; i += blockDim.x)
    if (sh[i]) atomicAdd(&hist[i], sh[i]);
}
__global__ void k_csel_compact(const double* keys, const Raw* in, unsigned n, const SelState* st, Raw* out, unsigned* count,
                               unsigned cap) {
  double thr = __longlong_as_double((long long)st->thresh);
  thr = st->takeall ? 0.0 : thr * (1.0 - 1e-12);
  for (unsigned t = blockIdx.x * blockDim.x + threadIdx.x; t < n; t += gridDim.x * blockDim.x) {
    if (keys[t] >= thr) {
      unsigned idx = atomicAdd(count, 1u);
      if (idx < cap) out[idx] = in[t];
    }
  }
}
// exact scores of the collected candidates:  logp_m + log(u / Z_m)
__global__ void k_sel_score(SelArgs a, const Raw* raw, unsigned n, unsigned npad, const double* logp, const double* Z,
                            int ns, int S, Cand* out) {
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= npad) return;
  if (t >= n) { out[t] = Cand{-INFINITY, 0x7fffffff, 0xffffffffu}; return; }
  Raw q = raw[t];
  int b = q.i / a.nCl, cl = q.i % a.nCl;
  double u = a.V[(i64)q.m * a.per_m + (i64)q.i * a.nA + q.a] * sel_fcd(a, q.m, cl, q.ch);
  unsigned state = (unsigned)q.a;
  if (S >= 2) state |= (unsigned)b << ns;
  if (S == 3) state |= ((unsigned)cl | ((unsigned)q.ch << (ns / 2))) << (2 * ns);
  out[t] = Cand{logp[q.m] + log(u / Z[q.m]), q.m, state};
}
__device__ __forceinline__ bool cand_before(const Cand& x, const Cand& y) {   // reading S8 total order
  if (x.score != y.score) return x.score > y.score;
  if (x.parent != y.parent) return x.parent < y.parent;
  return x.state < y.state;
}
__global__ void __launch_bounds__(1024) k_bitonic_smem(Cand* c, unsigned n) {
  extern __shared__ Cand sc[];
  for (unsigned i = threadIdx.x; i < n; i += blockDim.x) sc[i] = c[i];
  __syncthreads();
  for (unsigned k = 2; k <= n; k <<= 1)
    for (unsigned j = k >> 1; j > 0; j >>= 1) {
      for (unsigned i = threadIdx.x; i < n; i += blockDim.x) {
        unsigned l = i ^ j;
        if (l > i) {
          Cand x = sc[i], y = sc[l];
          bool up = (i & k) == 0;
          if (up ? cand_before(y, x) : cand_before(x, y)) { sc[i] = y; sc[l] = x; }
        }
      }
      __syncthreads();
    }
  for (unsigned i = threadIdx.x; i < n; i += blockDim.x) c[i] = sc[i];
}
// ---- merge by boundary (Fig. 3(d), Eq. (8)) ------------------------------------------
// Candidates with the same boundary (the projected legs of visited cells towards not yet visited cells) have
// identical futures; only the most probable one is kept.  The boundary of candidate (m, a, b, c_lo, c_hi) is
// (pid[m], P_right a, P_down b, P_dout c_lo): c_hi never appears (its only neighbour, up-left, is visited), so the
// prefilter already keeps one c_hi per V entry; pid[m] = dense id of the parent's part (host, from the beam states).
struct MCand { unsigned long long g; double score; int parent; unsigned state; };
__device__ __forceinline__ bool mcand_before(const MCand& x, const MCand& y) {
  if (x.g != y.g) return x.g < y.g;
  if (x.score != y.score) return x.score > y.score;
  if (x.parent != y.parent) return x.parent < y.parent;
  return x.state < y.state;
}
struct MergeLegs { const int *Pr, *Pd, *Po; int n_r, n_d, n_o, use_r, use_d, use_o; };
__device__ __forceinline__ unsigned long long merge_gid(const MergeLegs& lg, const int* pid, int m, int a, int b, int cl) {
  unsigned long long g = (unsigned long long)pid[m];
  g = g * (unsigned long long)(lg.use_r ? lg.n_r : 1) + (unsigned long long)(lg.use_r ? lg.Pr[a] : 0);
  g = g * (unsigned long long)(lg.use_d ? lg.n_d : 1) + (unsigned long long)(lg.use_d ? lg.Pd[b] : 0);
  g = g * (unsigned long long)(lg.use_o ? lg.n_o : 1) + (unsigned long long)(lg.use_o ? lg.Po[cl] : 0);
  return g;
}
// Droplet mode (TN_OPT_DROPLETS): every c_hi variant at or above the bound is a candidate (the interior variants are
// the losers that become droplets), and with `gbest` the bound is per boundary group: dfac x the group's best key.
__global__ void __launch_bounds__(256) k_sel_prefilter_all(SelArgs a, int lgA, int lgCl, double thr, double dfac,
                                                           const unsigned long long* gbest, const int* pid, MergeLegs lg,
                                                           Raw* out, unsigned* count, unsigned cap) {
  const int m = blockIdx.y, nchunk = gridDim.x;
  const i64 c0 = a.per_m * blockIdx.x / nchunk, c1 = a.per_m * (blockIdx.x + 1) / nchunk;
  const double* v = a.V + (i64)m * a.per_m;
  const double sc = a.scale[m];
  for (i64 q = c0 + threadIdx.x; q < c1; q += 256) {
    const double x = v[q];
    if (!(x > 0.0)) continue;
    const int i = (int)(q >> lgA), aa = (int)(q & (a.nA - 1)), cl = i & (a.nCl - 1), b = i >> lgCl;
    double bound = thr;
    if (gbest) bound = __longlong_as_double((long long)gbest[merge_gid(lg, pid, m, aa, b, cl)]) * dfac * (1.0 - 1e-12);
    const double vs = x * sc;
    for (int ch = 0; ch < a.nCh; ch++) {
      const double r = vs * sel_fcd(a, m, cl, ch);
      if (r > 0.0 && r >= bound) {
        unsigned idx = atomicAdd(count, 1u);
        if (idx < cap) out[idx] = Raw{m, i, aa, ch};
      }
    }
  }
}
__global__ void __launch_bounds__(256) k_sel_prefilter_merge(SelArgs a, int lgA, double thr, const double* fmx, Raw* out,
                                                             unsigned* count, unsigned cap) {
  const int m = blockIdx.y, nchunk = gridDim.x;
  const i64 per2 = a.per_m >> 1;
  const i64 c0 = per2 * blockIdx.x / nchunk, c1 = per2 * (blockIdx.x + 1) / nchunk;
  const double2* v2 = reinterpret_cast<const double2*>(a.V + (i64)m * a.per_m);
  const double sc = a.scale[m];
  const double* fm = fmx + (i64)m * a.nCl;
  for (i64 q = c0 + threadIdx.x; q < c1; q += 256) {
    const double2 x = v2[q];
    const int i = (int)((2 * q) >> lgA), cl = i & (a.nCl - 1);
    const double bound = fmax(x.x, x.y) * sc * fm[cl];
    if (!(bound >= thr) || !(bound > 0.0)) continue;
#pragma unroll
    for (int e = 0; e < 2; e++) {
      const double v = e ? x.y : x.x;
      if (!(v > 0.0) || !(v * sc * fm[cl] >= thr)) continue;
      int best = 0;
      double rb = -1.0;
      for (int ch = 0; ch < a.nCh; ch++) {
        const double r = sel_fcd(a, m, cl, ch);
        if (r > rb) { rb = r; best = ch; }
      }
      if (!(rb > 0.0)) continue;
      unsigned idx = atomicAdd(count, 1u);
      if (idx < cap) out[idx] = Raw{m, i, (int)((2 * q + e) & (a.nA - 1)), best};
    }
  }
}
__global__ void k_merge_score(SelArgs a, const Raw* raw, unsigned n, unsigned npad, const double* logp, const double* Z,
                              int ns, int S, const int* pid, MergeLegs lg, MCand* out) {
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= npad) return;
  if (t >= n) { out[t] = MCand{~0ull, -INFINITY, 0x7fffffff, 0xffffffffu}; return; }
  Raw q = raw[t];
  int b = q.i / a.nCl, cl = q.i % a.nCl;
  double u = a.V[(i64)q.m * a.per_m + (i64)q.i * a.nA + q.a] * sel_fcd(a, q.m, cl, q.ch);
  unsigned state = (unsigned)q.a;
  if (S >= 2) state |= (unsigned)b << ns;
  if (S == 3) state |= ((unsigned)cl | ((unsigned)q.ch << (ns / 2))) << (2 * ns);
  // for S == 1 the vertical sub-cluster IS sub-cluster 0: b == a there (i = b * nCl + cl with nCl = 1)
  unsigned long long g = (unsigned long long)pid[q.m];
  g = g * (unsigned long long)(lg.use_r ? lg.n_r : 1) + (unsigned long long)(lg.use_r ? lg.Pr[q.a] : 0);
  g = g * (unsigned long long)(lg.use_d ? lg.n_d : 1) + (unsigned long long)(lg.use_d ? lg.Pd[b] : 0);
  g = g * (unsigned long long)(lg.use_o ? lg.n_o : 1) + (unsigned long long)(lg.use_o ? lg.Po[cl] : 0);
  out[t] = MCand{g, logp[q.m] + log(u / Z[q.m]), q.m, state};
}
// ---- direct route when the number of POSSIBLE boundaries is small (last column / last row, small cells): a segmented
// arg-max over ALL entries of V keyed by the boundary id, with no threshold.  Pass 1: 64-bit atomicMax of the key bits
// of r = v * scale_m * max_ch fcd (positive doubles order like integers; r is monotone in the score); pass 2: among
// the entries that attain the maximum of their group, atomicMin of (parent << 32 | cell state) = the S8 tie-break;
// pass 3: one candidate per non-empty group with its exact score.
__device__ __forceinline__ unsigned merge_state(int a, int b, int cl, int ch, int ns, int S) {
  unsigned state = (unsigned)a;
  if (S >= 2) state |= (unsigned)b << ns;
  if (S == 3) state |= ((unsigned)cl | ((unsigned)ch << (ns / 2))) << (2 * ns);
  return state;
}
template <int PASS>
__global__ void __launch_bounds__(256) k_merge_seg(SelArgs a, int lgA, int lgCl, const double* fmx, const int* chbest,
                                                   const int* pid, MergeLegs lg, int ns, int S, unsigned long long* gbest,
                                                   unsigned long long* gtie, unsigned long long* npos) {
  const int m = blockIdx.y, nchunk = gridDim.x;
  const i64 c0 = a.per_m * blockIdx.x / nchunk, c1 = a.per_m * (blockIdx.x + 1) / nchunk;
  const double* v = a.V + (i64)m * a.per_m;
  const double sc = a.scale[m];
  unsigned cnt = 0;
  for (i64 q = c0 + threadIdx.x; q < c1; q += 256) {
    const double x = v[q];
    if (!(x > 0.0)) continue;
    const int i = (int)(q >> lgA), aa = (int)(q & (a.nA - 1)), cl = i & (a.nCl - 1), b = i >> lgCl;   // S == 1: X is the identity, positive entries have b == a
    const double r = x * sc * fmx[(i64)m * a.nCl + cl];
    if (!(r > 0.0)) continue;
    const unsigned long long key = (unsigned long long)__double_as_longlong(r);
    const unsigned long long g = merge_gid(lg, pid, m, aa, b, cl);
    if (PASS == 1) {
      atomicMax(&gbest[g], key);
      cnt++;
    } else if (gbest[g] == key) {
      const unsigned st = merge_state(aa, b, cl, chbest[(i64)m * a.nCl + cl], ns, S);
      atomicMin(&gtie[g], ((unsigned long long)m << 32) | st);
    }
  }
  if (PASS == 1 && cnt) atomicAdd(npos, (unsigned long long)cnt);
}
__global__ void k_merge_seg_emit(SelArgs a, const unsigned long long* gbest, const unsigned long long* gtie, i64 ngroups,
                                 const double* logp, const double* Z, int ns, int S, Cand* out, unsigned* count) {
  const i64 g = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= ngroups || gbest[g] == 0ull) return;
  const unsigned long long t = gtie[g];
  const int m = (int)(t >> 32);
  const unsigned st = (unsigned)(t & 0xffffffffull);
  const unsigned smask = (1u << ns) - 1, hmask = (1u << (ns / 2)) - 1;
  const int aa = (int)(st & smask), b = S == 1 ? aa : (int)((st >> ns) & smask);
  const int cl = S == 3 ? (int)((st >> (2 * ns)) & hmask) : 0, ch = S == 3 ? (int)((st >> (2 * ns + ns / 2)) & hmask) : 0;
  const int i = S == 1 ? aa : b * a.nCl + cl;
  const double u = a.V[(i64)m * a.per_m + (i64)i * a.nA + aa] * sel_fcd(a, m, cl, ch);
  out[atomicAdd(count, 1u)] = Cand{logp[m] + log(u / Z[m]), m, st};
}

// Bitonic sort of n = 2^p elements with shared-memory tiles of TILE elements: one launch sorts every tile up to
// k = TILE (direction from the GLOBAL index), then each k > TILE costs one global launch per j >= TILE and one
// launch that finishes j < TILE inside the tiles: 6 launches for 32768 elements instead of 120.
struct LessM { __device__ bool operator()(const MCand& x, const MCand& y) const { return mcand_before(x, y); } };
struct LessC { __device__ bool operator()(const Cand& x, const Cand& y) const { return cand_before(x, y); } };
template <class T, class Less, int TILE>
__global__ void __launch_bounds__(1024) k_bitonic_tile(T* c, unsigned n, unsigned kfirst, unsigned klast) {
  extern __shared__ unsigned char tile_raw[];
  T* sm = reinterpret_cast<T*>(tile_raw);
  const unsigned base = blockIdx.x * TILE, cnt = min((unsigned)TILE, n - base);
  Less less;
  for (unsigned i = threadIdx.x; i < cnt; i += blockDim.x) sm[i] = c[base + i];
  __syncthreads();
  for (unsigned k = kfirst; k <= klast; k <<= 1)
    for (unsigned j = min(k >> 1, (unsigned)TILE >> 1); j > 0; j >>= 1) {
      for (unsigned i = threadIdx.x; i < cnt; i += blockDim.x) {
        unsigned l = i ^ j;
        if (l > i) {
          T x = sm[i], y = sm[l];
          bool up = ((base + i) & k) == 0;
          if (up ? less(y, x) : less(x, y)) { sm[i] = y; sm[l] = x; }
        }
      }
      __syncthreads();
    }
  for (unsigned i = threadIdx.x; i < cnt; i += blockDim.x) c[base + i] = sm[i];
}
template <class T, class Less>
__global__ void k_bitonic_gstep(T* c, unsigned n, unsigned k, unsigned j) {
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  unsigned l = i ^ j;
  if (l > i) {
    Less less;
    T x = c[i], y = c[l];
    bool up = (i & k) == 0;
    if (up ? less(y, x) : less(x, y)) { c[i] = y; c[l] = x; }
  }
}
template <class T, class Less>
static void bitonic_sort(tn_handle* h, T* c, unsigned n) {   // n a power of two
  constexpr int TILE = 4096;
  TN_SMEM_OPT_IN(h, (k_bitonic_tile<T, Less, TILE>), TILE * (int)sizeof(T));
  const unsigned tiles = (n + TILE - 1) / TILE;
  k_bitonic_tile<T, Less, TILE><<<tiles, 1024, std::min<unsigned>(n, TILE) * sizeof(T), h->stream>>>(c, n, 2, std::min<unsigned>(n, TILE));
  TN_LAUNCH_CHECK(h);
  for (unsigned k = 2 * TILE; k <= n; k <<= 1) {
    for (unsigned j = k >> 1; j >= (unsigned)TILE; j >>= 1) {
      k_bitonic_gstep<T, Less><<<cdiv(n, 256), 256, 0, h->stream>>>(c, n, k, j);
      TN_LAUNCH_CHECK(h);
    }
    k_bitonic_tile<T, Less, TILE><<<tiles, 1024, TILE * sizeof(T), h->stream>>>(c, n, k, k);
    TN_LAUNCH_CHECK(h);
  }
}

// first (= most probable, S8 order) member of every group of the sorted list
__global__ void k_merge_first(const MCand* c, unsigned n, Cand* out, unsigned* count, double sthr = -INFINITY,
                              unsigned* count_thr = nullptr) {
  unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const MCand x = c[t];
  if (x.g == ~0ull) return;
  if (t == 0 || c[t - 1].g != x.g) {
    out[atomicAdd(count, 1u)] = Cand{x.score, x.parent, x.state};
    if (count_thr && x.score >= sthr) atomicAdd(count_thr, 1u);   // winners at or above the selection bound itself
  }
}

// ---- droplets (Fig. 4; reading S24) ---------------------------------------------------------
// One CTA per new beam element i (= kept winner of a boundary group).  Candidates: the droplets its parent carries,
// then every loser of its group within max_dE (sorted list `mc`: groups contiguous, S8 order inside), each followed by
// its compositions with the droplets of the loser's parent.  They are sorted by (dE, generation order) and kept
// greedily iff the flipped spins are one connected piece of the interaction graph and the Hamming distance to every
// droplet already kept is >= min_hamming, up to max_count.
struct DropArgs {
  const MCand* mc; unsigned n_mc;                 // sorted survivors of this cell's merge
  const Cand* beam; int nkeep;                    // new beam (sorted): parent, state, score
  const unsigned* st_old; int ncell, cellidx;     // old beam states
  const int* pid; MergeLegs lg; int ns, S, nCl;
  const unsigned* pool_old; const double* dE_old; const int* cnt_old;   // [m][K][ncell], [m][K], [m]
  unsigned* pool_new; double* dE_new; int* cnt_new;
  int K; double max_dE, beta; int min_hamming;
  const int* spin_of; int nbits;                  // [ncell][nbits]
  const int *adj_ptr, *adj; int n_spins;
  unsigned long long* overflow;
};
struct DCand { double dE; int seq, lparent, ldrop; unsigned lstate; };
constexpr int DROP_CMAX = 1024;
__global__ void __launch_bounds__(128) k_droplets(DropArgs a) {
  extern __shared__ unsigned char dsm_raw[];
  DCand* cand = reinterpret_cast<DCand*>(dsm_raw);                       // DROP_CMAX
  unsigned* fm = reinterpret_cast<unsigned*>(cand + DROP_CMAX);          // ncell
  unsigned* inF = fm + a.ncell;                                          // (n_spins + 31) / 32
  unsigned* reach = inF + (a.n_spins + 31) / 32;
  int* list = reinterpret_cast<int*>(reach + (a.n_spins + 31) / 32);     // n_spins
  __shared__ int s_n, s_scan[128], s_stop, s_cnt, s_changed, s_red[128];
  const int i = blockIdx.x, tid = threadIdx.x;
  const Cand w = a.beam[i];
  const unsigned smask = (1u << a.ns) - 1, hmask = (1u << (a.ns / 2)) - 1;
  const int wa = (int)(w.state & smask), wb = a.S == 1 ? wa : (int)((w.state >> a.ns) & smask);
  const int wcl = a.S == 3 ? (int)((w.state >> (2 * a.ns)) & hmask) : 0;
  const unsigned long long gw = merge_gid(a.lg, a.pid, w.parent, wa, wb, wcl);
  // group start: lower bound of gw in the sorted list (the winner itself is the first entry of its group)
  unsigned lo = 0, hi = a.n_mc;
  while (lo < hi) { unsigned mid = (lo + hi) >> 1; if (a.mc[mid].g < gw) lo = mid + 1; else hi = mid; }
  // ---- candidates, in generation order: inherited, then every loser followed by its compositions
  const int nin = a.cnt_old[w.parent];
  for (int k = tid; k < nin; k += 128) cand[k] = DCand{a.dE_old[(i64)w.parent * a.K + k], k, -1, k, 0u};
  if (tid == 0) { s_n = nin; s_stop = 0; }
  __syncthreads();
  for (unsigned base = lo + 1; !s_stop; base += 128) {
    const unsigned t = base + tid;
    int mine = 0;
    double dE = 0.0;
    MCand l;
    bool valid = false;
    if (t < a.n_mc) {
      l = a.mc[t];
      if (l.g == gw) {
        dE = (w.score - l.score) / a.beta;
        valid = dE <= a.max_dE;                     // sorted by score: the first loser beyond the cutoff ends the walk
      }
    }
    if (valid) {
      mine = 1;
      const int nl = a.cnt_old[l.parent];
      for (int k = 0; k < nl; k++) mine += (dE + a.dE_old[(i64)l.parent * a.K + k] <= a.max_dE) ? 1 : 0;
    }
    s_scan[tid] = mine;
    __syncthreads();
    if (tid == 0) {
      int run = s_n;
      bool stop = false;
      for (int q = 0; q < 128; q++) { const int c = s_scan[q]; s_scan[q] = run; run += c; if (c == 0) stop = true; }
      s_n = run;
      if (stop) s_stop = 1;
    }
    __syncthreads();
    if (valid) {
      int o = s_scan[tid];
      if (o < DROP_CMAX) cand[o] = DCand{dE, o, l.parent, -1, l.state};
      o++;
      const int nl = a.cnt_old[l.parent];
      for (int k = 0; k < nl; k++) {
        const double d2 = dE + a.dE_old[(i64)l.parent * a.K + k];
        if (d2 <= a.max_dE) { if (o < DROP_CMAX) cand[o] = DCand{d2, o, l.parent, k, l.state}; o++; }
      }
    }
    __syncthreads();
  }
  int n = s_n;
  if (n > DROP_CMAX) { if (tid == 0) atomicAdd(a.overflow, 1ull); n = DROP_CMAX; }
  int np2 = 1;
  while (np2 < n) np2 <<= 1;
  for (int k = n + tid; k < np2; k += 128) cand[k] = DCand{INFINITY, 0x7fffffff, -1, -1, 0u};
  __syncthreads();
  for (int k = 2; k <= np2; k <<= 1)                 // bitonic sort by (dE, generation order)
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int e = tid; e < np2; e += 128) {
        const int o = e ^ j;
        if (o > e) {
          const DCand x = cand[e], y = cand[o];
          const bool xy = x.dE < y.dE || (x.dE == y.dE && x.seq < y.seq);   // x before y
          const bool up = (e & k) == 0;
          if (up ? !xy : xy) { cand[e] = y; cand[o] = x; }
        }
      }
      __syncthreads();
    }
  // ---- greedy selection.  Every value that thread 0 publishes through s_cnt is copied to a register by all threads
  // and followed by a barrier before s_cnt is reused (the control flow below must stay uniform over the CTA).
  const int nw = (a.n_spins + 31) / 32;
  int kept = 0;
  unsigned* mine_pool = a.pool_new + (i64)i * a.K * a.ncell;
  for (int c = 0; c < n && kept < a.K; c++) {
    const DCand d = cand[c];
    // flip mask over cells
    int pop = 0;
    for (int k = tid; k < a.ncell; k += 128) {
      unsigned v = 0u;
      if (k <= a.cellidx) {
        if (d.lparent >= 0) {
          v = k < a.cellidx ? (a.st_old[(i64)d.lparent * a.ncell + k] ^ a.st_old[(i64)w.parent * a.ncell + k])
                            : (d.lstate ^ w.state);
        }
        if (d.ldrop >= 0) v ^= a.pool_old[((i64)(d.lparent >= 0 ? d.lparent : w.parent) * a.K + d.ldrop) * a.ncell + k];
      }
      fm[k] = v;
      pop += __popc(v);
    }
    s_red[tid] = pop;
    for (int k = tid; k < nw; k += 128) { inF[k] = 0u; reach[k] = 0u; }
    __syncthreads();
    if (tid == 0) { int t = 0; for (int q = 0; q < 128; q++) t += s_red[q]; s_cnt = t; }
    __syncthreads();
    const int nflip = s_cnt;
    __syncthreads();
    if (nflip == 0) continue;
    // Hamming distance to the kept ones
    bool ok = true;
    for (int j = 0; j < kept && ok; j++) {
      int hd = 0;
      for (int k = tid; k < a.ncell; k += 128) hd += __popc(fm[k] ^ mine_pool[(i64)j * a.ncell + k]);
      s_red[tid] = hd;
      __syncthreads();
      if (tid == 0) { int t = 0; for (int q = 0; q < 128; q++) t += s_red[q]; s_cnt = t; }
      __syncthreads();
      const int hdist = s_cnt;
      __syncthreads();
      if (hdist < a.min_hamming) ok = false;
    }
    if (ok) {
      // connectivity: list of flipped spins, label propagation from the lowest one
      if (tid == 0) s_cnt = 0;
      __syncthreads();
      for (int k = tid; k < a.ncell; k += 128) {
        unsigned v = fm[k];
        while (v) {
          const int bit = __ffs(v) - 1;
          v &= v - 1;
          const int sp = a.spin_of[k * a.nbits + bit];
          list[atomicAdd(&s_cnt, 1)] = sp;
          atomicOr(&inF[sp >> 5], 1u << (sp & 31));
        }
      }
      __syncthreads();
      if (tid == 0) { int mn = list[0]; for (int q = 1; q < nflip; q++) mn = min(mn, list[q]); reach[mn >> 5] |= 1u << (mn & 31); }
      __syncthreads();
      for (int round = 0; round < nflip; round++) {
        if (tid == 0) s_changed = 0;
        __syncthreads();
        for (int q = tid; q < nflip; q += 128) {
          const int u = list[q];
          if (!((reach[u >> 5] >> (u & 31)) & 1u)) continue;
          for (int e = a.adj_ptr[u]; e < a.adj_ptr[u + 1]; e++) {
            const int v = a.adj[e];
            if (((inF[v >> 5] >> (v & 31)) & 1u) && !((reach[v >> 5] >> (v & 31)) & 1u)) {
              atomicOr(&reach[v >> 5], 1u << (v & 31));
              s_changed = 1;
            }
          }
        }
        __syncthreads();
        const int ch = s_changed;
        __syncthreads();
        if (!ch) break;
      }
      int rc = 0;
      for (int k = tid; k < nw; k += 128) rc += __popc(reach[k]);
      s_red[tid] = rc;
      __syncthreads();
      if (tid == 0) { int t = 0; for (int q = 0; q < 128; q++) t += s_red[q]; s_cnt = t; }
      __syncthreads();
      const int nreach = s_cnt;
      __syncthreads();
      if (nreach != nflip) ok = false;
    }
    if (ok) {
      for (int k = tid; k < a.ncell; k += 128) mine_pool[(i64)kept * a.ncell + k] = fm[k];
      if (tid == 0) a.dE_new[(i64)i * a.K + kept] = d.dE;
      kept++;
    }
    __syncthreads();
  }
  if (tid == 0) a.cnt_new[i] = kept;
}
// cells selected without merging: the children inherit their parent's droplets unchanged
__global__ void k_droplets_inherit(const Cand* beam, int nkeep, int K, int ncell, const unsigned* pool_old, const double* dE_old,
                                   const int* cnt_old, unsigned* pool_new, double* dE_new, int* cnt_new) {
  const int i = blockIdx.x, p = beam[i].parent, n = cnt_old[p];
  for (i64 k = threadIdx.x; k < (i64)n * ncell; k += blockDim.x) pool_new[(i64)i * K * ncell + k] = pool_old[(i64)p * K * ncell + k];
  for (int k = threadIdx.x; k < n; k += blockDim.x) dE_new[(i64)i * K + k] = dE_old[(i64)p * K + k];
  if (threadIdx.x == 0) cnt_new[i] = n;
}
// flips[(i, k)][spin] = 1 if droplet k of state i flips that spin
__global__ void k_droplets_unpack(const unsigned* pool, int nstate, int K, int ncell, int n_spins, const int* cell_of,
                                  const int* bit_of, int8_t* out) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (i64)nstate * K * n_spins) return;
  const int sp = (int)(t % n_spins);
  const i64 ik = t / n_spins;
  out[t] = (int8_t)((pool[ik * ncell + cell_of[sp]] >> bit_of[sp]) & 1u);
}
__global__ void k_fill_sentinel(Cand* c, unsigned from, unsigned to) {
  unsigned t = from + blockIdx.x * blockDim.x + threadIdx.x;
  if (t < to) c[t] = Cand{-INFINITY, 0x7fffffff, 0xffffffffu};
}
static int pext_host(int v, int mask) {
  int out = 0, bit = 0;
  for (int i = 0; i < 8; i++)
    if ((mask >> i) & 1) { out |= ((v >> i) & 1) << bit; bit++; }
  return out;
}

// new beam from the sorted candidates
__global__ void k_new_beam(const Cand* cand, int nkeep, int M, const unsigned* st_old, unsigned* st_new, int ncell_ld,
                           int cellidx, const int* slot_old, int* slot_new, double* logp_new, const double* LG,
                           int npp, int Dr, int ldLv, double* Lv_new, const int* Pd, const int* Po, int n_o, int ns,
                           int S, double* pd_out) {
  int i = blockIdx.x;
  if (i >= nkeep) return;
  Cand c = cand[i];
  for (int k = threadIdx.x; k < cellidx; k += blockDim.x)
    st_new[(i64)i * ncell_ld + k] = st_old[(i64)c.parent * ncell_ld + k];
  __shared__ double sh[128];
  const int half = ns / 2;
  int b = S == 1 ? (c.state & ((1u << ns) - 1)) : ((c.state >> ns) & ((1u << ns) - 1));
  int cl = S == 3 ? ((c.state >> (2 * ns)) & ((1u << half) - 1)) : 0;
  const double* src = LG + ((i64)c.parent * npp + Pd[b] * n_o + Po[cl]) * Dr;
  double mx = 0.0;
  for (int k = threadIdx.x; k < Dr; k += blockDim.x) mx = fmax(mx, fabs(src[k]));
  sh[threadIdx.x] = mx;
  __syncthreads();
  for (int o = 64; o > 0; o >>= 1) {
    if (threadIdx.x < o) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + o]);
    __syncthreads();
  }
  mx = sh[0];
  for (int k = threadIdx.x; k < ldLv; k += blockDim.x)
    Lv_new[(i64)i * ldLv + k] = (k < Dr && mx > 0.0) ? src[k] / mx : 0.0;
  if (threadIdx.x == 0) {
    st_new[(i64)i * ncell_ld + cellidx] = c.state;
    slot_new[i] = slot_old[c.parent];
    logp_new[i] = c.score;
    if (i == 0 && pd_out) *pd_out = fmax(*pd_out, cand[M].score);   // cand padded: -inf when nothing was discarded
  }
}
__global__ void k_iota(int* p, int n) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = i;
}
__global__ void k_reset_lv(double* Lv, int nb, int ld) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < nb * ld) Lv[i] = (i % ld == 0) ? 1.0 : 0.0;
}
// unpack cell states to +-1 spins (spin-id order)
__global__ void k_unpack(const unsigned* states, int ncell_ld, int n, int n_spins, const int* cell_of, const int* bit_of,
                         int8_t* out) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (i64)n * n_spins) return;
  int m = (int)(t / n_spins), i = (int)(t % n_spins);
  unsigned st = states[(i64)m * ncell_ld + cell_of[i]];
  out[t] = (int8_t)(1 - 2 * (int)((st >> bit_of[i]) & 1u));
}
// O-0 energy: one running fp64 sum, edges in input order, then fields in spin order (Eq. (1))
__global__ void k_energy(const int8_t* s, int n, int n_spins, i64 n_edges, const int* eu, const int* ev, const double* J,
                         const double* hf, double* E) {
  int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n) return;
  const int8_t* sm = s + (i64)m * n_spins;
  double e = 0.0;
  for (i64 k = 0; k < n_edges; k++) e = e + J[k] * (double)((int)sm[eu[k]] * (int)sm[ev[k]]);
  for (int i = 0; i < n_spins; i++) e = e + hf[i] * (double)sm[i];
  E[m] = e;
}

template <class T>
T d2h(tn_handle* h, const T* p) {
  T v;
  TN_CUDA(cudaMemcpyAsync(&v, p, sizeof(T), cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaStreamSynchronize(h->stream));
  return v;
}

struct Tic {
  tn_handle* h; double* dst; cudaEvent_t a = nullptr, b = nullptr;
  Tic(tn_handle* h_, double* d) : h(h_), dst(d) { cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, h->stream); }
  Tic(const Tic&) = delete;
  Tic& operator=(const Tic&) = delete;
  void stop() {
    cudaEventRecord(b, h->stream); cudaEventSynchronize(b);
    float ms = 0; if (cudaEventElapsedTime(&ms, a, b) == cudaSuccess) *dst += ms;
    cudaEventDestroy(a); cudaEventDestroy(b);
    a = b = nullptr;
  }
  ~Tic() {   // an exception between the constructor and stop(): the events do not outlive the call
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
  }
};

void build_G(tn_handle* h, const MpsTensor& S, const MpsTensor* Q, RowTab& rt) {
  if (Q) {
    rt.Dl = S.dl; rt.Dr = Q->dr; rt.npp = S.p * Q->p;
    rt.G = h->dalloc<double>((size_t)rt.npp * rt.Dl * rt.Dr);
    GemmDesc g;
    g.B1 = S.p; g.B2 = Q->p; g.M = S.dl; g.N = Q->dr; g.K = S.dr;
    g.A = S.d; g.a_b1 = S.dr; g.a_b2 = 0; g.a_i = (i64)S.p * S.dr; g.a_k = 1;
    g.B = Q->d; g.b_b1 = 0; g.b_b2 = Q->dr; g.b_k = (i64)Q->p * Q->dr; g.b_j = 1;
    g.C = rt.G; g.c_b1 = (i64)Q->p * rt.Dl * rt.Dr; g.c_b2 = (i64)rt.Dl * rt.Dr; g.c_i = rt.Dr; g.c_j = 1;
    g.nsplit = 1;
    gemm_general(h, g);
    h->st.flop_search += 2.0 * rt.npp * rt.Dl * (double)rt.Dr * S.dr;
    h->st.flop_search_rblocks += 2.0 * rt.npp * rt.Dl * (double)rt.Dr * S.dr;
  } else {
    rt.Dl = S.dl; rt.Dr = S.dr; rt.npp = S.p;
    rt.G = h->dalloc<double>((size_t)rt.npp * rt.Dl * rt.Dr);
    permute3(h, rt.G, S.d, S.p, S.dl, S.dr, S.dr, (i64)S.p * S.dr, 1);
  }
}

void run(tn_handle* h, int M, bool logz_only, int* n_out, int8_t* states_out, double* energies, double* logp_out,
         double* log_pd_out) {
  const int Ly = h->Ly, Lx = h->Lx, ns = h->ns, S = h->S, ncell = Ly * Lx;
  int Dmax = 1;
  for (int y = 1; y <= Ly; y++)
    for (auto& t : h->rows[y]) Dmax = std::max(Dmax, std::max(t.dl, t.dr));
  const int ldLv = Dmax;
  const unsigned cap = (unsigned)std::max(2 * (i64)M, (i64)M + 2048);
  unsigned npad = 4096;
  while (npad < cap) npad <<= 1;
  DBuf<unsigned> stA(h, (size_t)M * ncell), stB(h, (size_t)M * ncell);
  DBuf<double> lpA(h, M), lpB(h, M), LvA(h, (size_t)M * ldLv), LvB(h, (size_t)M * ldLv);
  DBuf<int> slA(h, M), slB(h, M), hrow(h, M), vrow(h, (size_t)M * Lx), drow(h, (size_t)M * Lx);
  DBuf<double> Z(h, M), scale(h, (size_t)M + 1), pd(h, 1), fc(h, (size_t)M * 16);
  DBuf<unsigned long long> nneg(h, 1);
  DBuf<SelState> sel(h, 1);
  DBuf<unsigned> hist(h, 4096), count(h, 2);
  DBuf<Raw> raw(h, cap);
  const unsigned ccap = 1u << 22;                   // compact candidate list of the prefilter pass
  DBuf<double> ckeys(h, ccap), fmx(h, (size_t)M * 16);
  DBuf<Raw> craw(h, ccap);
  const unsigned mcap = h->merge ? (unsigned)h->merge_cap : 1u;   // survivors / boundary groups handled by the merge route
  size_t mcap2 = 2;                                    // sort buffers: next power of two above max(mcap, M) entries
  while (mcap2 < (size_t)std::max<i64>(mcap, M) + 1) mcap2 <<= 1;
  DBuf<MCand> mcand(h, h->merge ? mcap2 : 1);
  DBuf<Cand> mcands(h, h->merge ? mcap2 + 4096 : 1);
  DBuf<int> pid(h, M), chbest(h, h->merge ? (size_t)M * 16 : 1);
  // ---- droplets (Fig. 4): double-buffered pools [beam element][K][cell] of xor masks, their dE and counts
  const bool drops = h->merge && h->droplets;
  const int dK = drops ? h->droplet_max_count : 1, nbits = S * ns;
  const size_t dpool = drops ? (size_t)M * dK * ncell : 1;
  DBuf<unsigned> dpA(h, dpool), dpB(h, dpool);
  DBuf<double> ddA(h, (size_t)M * dK), ddB(h, (size_t)M * dK);
  DBuf<int> dcA(h, M), dcB(h, M), d_spin_of(h, drops ? (size_t)ncell * nbits : 1), d_adj_ptr(h, drops ? (size_t)h->n_spins + 1 : 1);
  DBuf<int> d_adj(h, drops ? 2 * (size_t)h->n_edges + 1 : 1);
  DBuf<unsigned long long> d_dover(h, 1);
  unsigned* dp_cur = dpA.p; unsigned* dp_nxt = dpB.p;
  double* dd_cur = ddA.p; double* dd_nxt = ddB.p;
  int* dc_cur = dcA.p; int* dc_nxt = dcB.p;
  size_t drop_smem = 0;
  if (drops) {
    if (h->n_spins > 16384) tn_throw(TN_ERR_ARG, "TN_OPT_DROPLETS supports up to 16384 spins");
    std::vector<int> spin_of((size_t)ncell * nbits, 0), aptr((size_t)h->n_spins + 1, 0), adj;
    for (int i = 0; i < h->n_spins; i++) spin_of[(size_t)h->cell_of[i] * nbits + h->bit_of[i]] = i;
    for (i64 e = 0; e < h->n_edges; e++)
      if (h->J[e] != 0.0) { aptr[h->edge_u[e] + 1]++; aptr[h->edge_v[e] + 1]++; }
    for (int i = 0; i < h->n_spins; i++) aptr[i + 1] += aptr[i];
    adj.assign((size_t)aptr[h->n_spins] + 1, 0);
    std::vector<int> fill(aptr.begin(), aptr.end() - 1);
    for (i64 e = 0; e < h->n_edges; e++)
      if (h->J[e] != 0.0) { adj[fill[h->edge_u[e]]++] = h->edge_v[e]; adj[fill[h->edge_v[e]]++] = h->edge_u[e]; }
    TN_CUDA(cudaMemcpyAsync(d_spin_of.p, spin_of.data(), sizeof(int) * spin_of.size(), cudaMemcpyHostToDevice, h->stream));
    TN_CUDA(cudaMemcpyAsync(d_adj_ptr.p, aptr.data(), sizeof(int) * aptr.size(), cudaMemcpyHostToDevice, h->stream));
    TN_CUDA(cudaMemcpyAsync(d_adj.p, adj.data(), sizeof(int) * adj.size(), cudaMemcpyHostToDevice, h->stream));
    TN_CUDA(cudaMemsetAsync(dpA.p, 0, sizeof(unsigned) * dpool, h->stream));
    TN_CUDA(cudaMemsetAsync(dpB.p, 0, sizeof(unsigned) * dpool, h->stream));
    TN_CUDA(cudaMemsetAsync(dcA.p, 0, sizeof(int) * M, h->stream));
    TN_CUDA(cudaMemsetAsync(d_dover.p, 0, sizeof(unsigned long long), h->stream));
    TN_CUDA(cudaStreamSynchronize(h->stream));   // the host vectors above go out of scope
    drop_smem = sizeof(DCand) * DROP_CMAX + sizeof(unsigned) * ((size_t)ncell + 2 * ((h->n_spins + 31) / 32)) +
                sizeof(int) * (size_t)h->n_spins;
    TN_SMEM_OPT_IN(h, k_droplets, 200 * 1024);
    if (drop_smem > 200 * 1024) tn_throw(TN_ERR_ARG, "TN_OPT_DROPLETS: lattice too large for the droplet kernel");
  }
  const double dfac = drops ? std::exp(-h->beta * h->droplet_max_dE) * (1.0 - 1e-9) : 1.0;
  DBuf<unsigned long long> gbest(h, 2 * (size_t)mcap + 2);   // [mcap] group maxima, [mcap] tie-breaks, [1] positive-entry count
  DBuf<Cand> cand(h, npad);
  unsigned* st_cur = stA.p; unsigned* st_nxt = stB.p;
  double* lp_cur = lpA.p; double* lp_nxt = lpB.p;
  double* Lv_cur = LvA.p; double* Lv_nxt = LvB.p;
  int* sl_cur = slA.p; int* sl_nxt = slB.p;
  int nb = 1;
  fill_value(h, lp_cur, 1, 0.0);
  fill_value(h, pd.p, 1, -INFINITY);
  TN_CUDA(cudaMemsetAsync(nneg.p, 0, sizeof(unsigned long long), h->stream));
  TN_CUDA(cudaMemsetAsync(hist.p, 0, sizeof(unsigned) * 4096, h->stream));
  TN_CUDA(cudaMemsetAsync(st_cur, 0, sizeof(unsigned) * ncell, h->stream));
  TN_SMEM_OPT_IN(h, k_bitonic_smem, 8192 * (int)sizeof(Cand));

  for (int y = 0; y < Ly; y++) {
    const std::vector<MpsTensor>& R = h->rows[y + 1];
    std::vector<RowTab> rt(Lx);
    const int nb_row = nb;   // beam size at the row start = number of right-block slots
    // ---- row start: tables of R_{y+1}, above-row indices, right blocks (a4 (ii))
    Tic t_rb(h, &h->st.ms_search_rblocks);
    for (int x = 0; x < Lx; x++) {
      rt[x].c = &h->cell(y, x);
      const MpsTensor& Sx = h->has_med() ? R[2 * x] : R[x];
      const MpsTensor* Qx = (h->has_med() && x + 1 < Lx) ? &R[2 * x + 1] : nullptr;
      build_G(h, Sx, Qx, rt[x]);
      rt[x].RM = h->dalloc<double>((size_t)nb * rt[x].Dr * rt[x].c->n_r);
      rt[x].ls = h->dalloc<double>(nb);
    }
    k_above_rows<<<cdiv((i64)nb * Lx, 256), 256, 0, h->stream>>>(st_cur, ncell, nb, y, Lx, ns, S, h->d_cells, vrow.p, drow.p);
    TN_LAUNCH_CHECK(h);
    k_iota<<<cdiv(nb, 256), 256, 0, h->stream>>>(sl_cur, nb);
    TN_LAUNCH_CHECK(h);
    k_reset_lv<<<cdiv((i64)nb * ldLv, 256), 256, 0, h->stream>>>(Lv_cur, nb, ldLv);
    TN_LAUNCH_CHECK(h);
    fill_value(h, rt[Lx - 1].RM, (i64)nb * rt[Lx - 1].Dr * rt[Lx - 1].c->n_r, 1.0);
    fill_value(h, rt[Lx - 1].ls, nb, 0.0);
    for (int x = Lx - 1; x >= 1; x--) {
      const CellDev& c = *rt[x].c;
      const int Dl = rt[x].Dl, Dr = rt[x].Dr;
      const i64 DD = (i64)Dl * Dr;
      DBuf<double> fcx(h, (size_t)nb * c.nCl), H(h, (size_t)nb * c.nT * DD), RS(h, (size_t)nb * Dl * c.nA);
      k_fc<<<cdiv((i64)nb * c.nCl, 256), 256, 0, h->stream>>>(c, drow.p + (size_t)x * nb, nullptr, nb, fcx.p);
      TN_LAUNCH_CHECK(h);
      {   // H[(m,t)][(b',b'')] = sum_{(b,cl)} coef[(b,cl)][(m,t)] G[(Pd b, Po cl)][(b',b'')]
        const int Mg = (int)DD, Ng = nb * c.nT, Kg = c.nB * c.nCl;
        bool done = false;
        const bool fact = h->rblock_fact && c.nT <= 16 && c.nCl <= 16;
        const double fl = fact ? 2.0 * Mg * (double)nb * c.nB * (c.nCl + c.nT) : 2.0 * Mg * (double)Ng * Kg;
        h->st.flop_search += fl;
        h->st.flop_search_rblocks += fl + 2.0 * nb * (double)Dl * c.nA * Dr + 2.0 * nb * (double)Dl * c.bh_rows * c.nA;
        if (fact) {
          DBuf<double> Gy(h, (size_t)Kg * DD);
          k_gather_Gy<<<cdiv((i64)Kg * DD, 256), 256, 0, h->stream>>>(rt[x].G, c.Yc, c.Pd, c.Po, c.nCl, c.n_o, DD, Kg, Gy.p);
          TN_LAUNCH_CHECK(h);
          dim3 grid((unsigned)cdiv(DD, 64), (unsigned)cdiv(nb, 8));
          const bool mma = h->rblock_fact != 2 && (DD & 1) == 0;     // 16-byte cp.async rows
          if (mma && c.nT <= 8)
            launch_rblock_mma<1>(h, grid, Gy.p, c.X, c.BvS, fcx.p, vrow.p + (size_t)x * nb, nb, c.nB, c.nCl, c.nT, DD, H.p);
          else if (mma)
            launch_rblock_mma<2>(h, grid, Gy.p, c.X, c.BvS, fcx.p, vrow.p + (size_t)x * nb, nb, c.nB, c.nCl, c.nT, DD, H.p);
          else if (c.nT <= 4)
            k_rblock_h<4><<<grid, 256, 0, h->stream>>>(Gy.p, c.X, c.BvS, fcx.p, vrow.p + (size_t)x * nb, nb, c.nB, c.nCl, c.nT, DD, H.p);
          else
            k_rblock_h<16><<<grid, 256, 0, h->stream>>>(Gy.p, c.X, c.BvS, fcx.p, vrow.p + (size_t)x * nb, nb, c.nB, c.nCl, c.nT, DD, H.p);
          TN_LAUNCH_CHECK(h);
          done = true;
        }
        if (!done && (DD & 1) == 0 && (Ng & 1) == 0) {
          // both operands materialised row-major in the reduction index, then the streaming GEMM (tsgemm.cu)
          DBuf<double> Gg(h, (size_t)Kg * DD), cf(h, (size_t)Kg * Ng);
          k_gather_G<<<cdiv((i64)Kg * DD, 256), 256, 0, h->stream>>>(rt[x].G, c.Pd, c.Po, c.nCl, c.n_o, DD, Kg, Gg.p);
          TN_LAUNCH_CHECK(h);
          k_coef<<<cdiv((i64)Kg * Ng, 256), 256, 0, h->stream>>>(c.X, c.BvS, c.Yc, fcx.p, vrow.p + (size_t)x * nb, c.nB, c.nCl,
                                                               c.nT, Kg, Ng, cf.p);
          TN_LAUNCH_CHECK(h);
          done = tsgemm(h, true, Kg, Mg, Ng, cf.p, Ng, Gg.p, DD, H.p, DD);
        }
        if (!done) {
          LdHA a{rt[x].G, c.Pd, c.Po, c.nCl, c.n_o, DD};
          LdHB b{c.X, c.BvS, c.Yc, fcx.p, vrow.p + (size_t)x * nb, c.nB, c.nCl, c.nT};
          StH e{H.p, DD};
          dim3 grid(1, cdiv(Mg, 64), cdiv(Ng, 64));
          k_gemm<64, 64, 16, 2, 2, false, true, LdHA, LdHB, StH><<<grid, 128, 0, h->stream>>>(Mg, Ng, Kg, 1, a, b, e);
          TN_LAUNCH_CHECK(h);
        }
      }
      {
        i64 total = (i64)nb * Dl * c.nA;
        k_rs<<<cdiv(total, 256), 256, 0, h->stream>>>(c, H.p, rt[x].RM, nb, Dl, Dr, RS.p);
        TN_LAUNCH_CHECK(h);
      }
      // RM_{x-1}[(m, b'), r] = sum_a RS[(m, b'), a] BhS[r, a]: the beam stacks along the rows -> one GEMM
      gemm_rm(h, false, true, nb * Dl, c.bh_rows, c.nA, RS.p, c.nA, c.BhS, c.nA, rt[x - 1].RM, c.bh_rows);
      k_norm_rm<<<nb, 256, 0, h->stream>>>(rt[x - 1].RM, Dl * c.bh_rows, rt[x].ls, rt[x - 1].ls);
      TN_LAUNCH_CHECK(h);
    }
    t_rb.stop();

    for (int x = 0; x < Lx; x++) {
      const int cellidx = y * Lx + x;
      const CellDev& c = *rt[x].c;
      const int Dl = rt[x].Dl, Dr = rt[x].Dr, npp = rt[x].npp;
      const i64 per_m = (i64)c.nB * c.nCl * c.nA;
      Tic t_c(h, &h->st.ms_search_cond);
      DBuf<double> LG(h, (size_t)nb * npp * Dr), V(h, (size_t)nb * per_m);
      DBuf<double> rowmax(h, (size_t)nb * c.nB * c.nCl);   // largest entry of every row of V (written by k_cond)
      bool have_rowmax = false;
      bool lazy_v = false;                                 // V not written by k_cond: k_cond_rows fills the rows the selection reads
      CondArgs ca_rows{};                                  // the conditional kernel's arguments, kept for that second kernel
      std::unique_ptr<DBuf<double>> RMc_keep;              // its dense operand stays alive until then
      k_hrow<<<cdiv(nb, 256), 256, 0, h->stream>>>(st_cur, ncell, nb, cellidx, x, ns, h->d_cells, hrow.p);
      TN_LAUNCH_CHECK(h);
      k_fc<<<cdiv((i64)nb * c.nCl, 256), 256, 0, h->stream>>>(c, drow.p + (size_t)x * nb_row, sl_cur, nb, fc.p);
      TN_LAUNCH_CHECK(h);
      {   // LG[m][pp][b''] = sum_b' Lv[m][b'] G[pp][b'][b'']
        LdLv a{Lv_cur, ldLv};
        LdGj b{rt[x].G, Dl, Dr};
        StPlain e{LG.p, (i64)npp * Dr};
        int Ng = npp * Dr;
        dim3 grid(1, cdiv(nb, 64), cdiv(Ng, 64));
        k_gemm<64, 64, 16, 2, 2, true, true, LdLv, LdGj, StPlain><<<grid, 128, 0, h->stream>>>(nb, Ng, Dl, 1, a, b, e);
        TN_LAUNCH_CHECK(h);
        h->st.flop_search += 2.0 * nb * (double)Ng * Dl;
        h->st.flop_search_cond += 2.0 * nb * (double)Ng * Dl;
      }
      {   // V[m][(b,cl)][a]
        int Mg = c.nB * c.nCl, Ng = c.nA;
        h->st.flop_search += 2.0 * nb * (double)Mg * Ng * Dr;
        h->st.flop_search_cond += 2.0 * nb * (double)Mg * Ng * Dr;
        h->st.bytes_search_cond += 8.0 * nb * (double)per_m;
        RMc_keep.reset(new DBuf<double>(h, (size_t)nb * Dr * c.nA));
        DBuf<double>& RMc = *RMc_keep;
        k_rmc<<<cdiv((i64)nb * Dr * c.nA, 256), 256, 0, h->stream>>>(rt[x].RM, sl_cur, c.Pr, c.BhS, c.wA, hrow.p, nb, Dr, c.n_r, c.nA, RMc.p);
        TN_LAUNCH_CHECK(h);
        ArPV ar{LG.p, c.Pd, c.Po, c.nCl, c.n_o, npp, Dr};
        LdPB be{RMc.p, Dr, c.nA};
        const int ntile = (Mg + 127) / 128;
        DBuf<double> zpart(h, (size_t)nb * std::max(ntile, 64));
        EpPV ep{V.p, c.X, c.BvS, c.Yc, fc.p, vrow.p + (size_t)x * nb_row, sl_cur, zpart.p, nneg.p,
                c.nA, c.nB, c.nCl, c.tshift, ntile, per_m};
        CondArgs ca{LG.p, c.Pd, c.Po, c.nCl, c.n_o, npp, Dr, RMc.p, c.nA, V.p, c.X, c.BvS, c.Yc, fc.p,
                    vrow.p + (size_t)x * nb_row, sl_cur, zpart.p, nneg.p, c.nB, c.tshift, ntile, Mg, per_m,
                    h->select_rows ? rowmax.p : nullptr, 1, 1};
        // lazy V: only on the route that reads V through the row test (no merge, no droplets, not the direct passes)
        lazy_v = h->lazy_v && h->select_rows && !h->merge && !h->droplets &&
                 (i64)nb * per_m * c.nCh > (i64)h->select_direct_max;
        ca.store = lazy_v ? 0 : 1;
        if (h->cond_pipe && launch_cond(h, nb, ca)) {
          have_rowmax = h->select_rows != 0;
          ca_rows = ca;
          if (lazy_v) h->st.bytes_search_cond += 8.0 * nb * ((double)npp * Dr + (double)Dr * c.nA + Mg) - 8.0 * nb * (double)per_m;
          k_beam_Z_final<<<cdiv(nb, 128), 128, 0, h->stream>>>(zpart.p, nb, ntile, Z.p);
          TN_LAUNCH_CHECK(h);
        } else if ((lazy_v = false, launch_bgemm<false>(h, nb, Mg, Ng, Dr, ar, be, ep))) {
          // Z and the negative count came out of the GEMM epilogue: no extra pass over V
          k_beam_Z_final<<<cdiv(nb, 128), 128, 0, h->stream>>>(zpart.p, nb, ntile, Z.p);
          TN_LAUNCH_CHECK(h);
        } else {
          lazy_v = false;
          LdPA a{LG.p, c.Pd, c.Po, c.nCl, c.n_o, npp, Dr};
          StPV e{V.p, c.BhS, c.wA, c.X, c.BvS, c.Yc, hrow.p, vrow.p + (size_t)x * nb_row, sl_cur, c.nA, c.nB, c.nCl, c.tshift, per_m};
          dim3 grid(nb, cdiv(Mg, 64), cdiv(Ng, 64));
          k_gemm<64, 64, 16, 2, 2, true, true, LdPA, LdPB, StPV><<<grid, 128, 0, h->stream>>>(Mg, Ng, Dr, 1, a, be, e);
          TN_LAUNCH_CHECK(h);
          int lgA = 0;
          while ((1 << lgA) < c.nA) lgA++;
          const int nchunk = (int)std::max<i64>(1, std::min<i64>(64, per_m / 8192));
          k_beam_Z<<<dim3(nchunk, nb), 256, 0, h->stream>>>(V.p, per_m, lgA, c.nCl, fc.p, zpart.p, nneg.p);
          TN_LAUNCH_CHECK(h);
          k_beam_Z_final<<<cdiv(nb, 128), 128, 0, h->stream>>>(zpart.p, nb, nchunk, Z.p);
          TN_LAUNCH_CHECK(h);
        }
      }
      t_c.stop();
      if (y == 0 && x == 0) {
        double z0 = d2h(h, Z.p), ls0 = d2h(h, rt[0].ls);
        if (!(z0 > 0.0) || !std::isfinite(z0)) tn_throw(TN_ERR_NUMERIC, "first-cell normaliser is %g", z0);
        double lz = -h->beta * h->offset + std::log(z0) + ls0;
        for (int yy = 1; yy < Ly; yy++) lz += h->lognorm[yy];
        if (!std::isfinite(lz)) tn_throw(TN_ERR_NUMERIC, "log Z = %g is not finite (beta * offset = %g)", lz, h->beta * h->offset);
        h->log_z = lz;
        h->have_logz = true;
        if (logz_only) {
          for (auto& r : rt) { h->dfree(r.G); h->dfree(r.RM); h->dfree(r.ls); }
          return;
        }
      }
      // ---- selection
      Tic t_s(h, &h->st.ms_search_select);
      k_beam_scale<<<1, 256, 0, h->stream>>>(lp_cur, Z.p, nb, scale.p);
      TN_LAUNCH_CHECK(h);
      SelArgs sa{V.p, scale.p, c.wC, c.Bd, drow.p + (size_t)x * nb_row, sl_cur, c.Pi, per_m, nb, c.nA, c.nCl, c.nCh, c.n_i};
      SelState s0;
      memset(&s0, 0, sizeof(s0));
      s0.want = (unsigned long long)M + 1;
      TN_CUDA(cudaMemcpyAsync(sel.p, &s0, sizeof(s0), cudaMemcpyHostToDevice, h->stream));
      const int shifts[6] = {52, 40, 28, 16, 4, 0}, nbitsv[6] = {12, 12, 12, 12, 12, 4};
      const i64 total = (i64)nb * per_m;
      const int gsel = (int)std::min<i64>((i64)h->sms * 8, (total + 255) / 256);
      unsigned ncand = 0;
      // Ties at the cut beyond the candidate list (degenerate instances: integer couplings, J = 0): up to tie_cap candidates
      // are collected completely and sorted, so that the S8 order decides and the result is reproducible run to run;
      // beyond that an arbitrary subset of the tie group is taken and the cell is counted in select_tie_dropped.
      const unsigned tie_cap = 1u << 24;
      std::unique_ptr<DBuf<Raw>> rawL;
      std::unique_ptr<DBuf<Cand>> candL;
      bool direct = total * c.nCh <= (i64)h->select_direct_max;       // few candidates: radix passes straight on V
      bool cand_sorted = false;                                       // set by the merge route (cand.p final and sorted)
      unsigned np2 = 2;
      unsigned n_mc = 0;   // entries of the sorted survivor list mcand of this cell (droplet mode)
      if (h->merge) {
        // ---- parent part of the boundary: dense ids of the projected forward legs of rows y-1, y (host, tiny)
        std::vector<unsigned> hst((size_t)nb * ncell);
        TN_CUDA(cudaMemcpyAsync(hst.data(), st_cur, sizeof(unsigned) * hst.size(), cudaMemcpyDeviceToHost, h->stream));
        TN_CUDA(cudaStreamSynchronize(h->stream));
        std::map<std::vector<int>, int> ids;
        std::vector<int> hpid(nb), key;
        const unsigned smask = (1u << ns) - 1, hmask = (1u << (ns / 2)) - 1;
        for (int m = 0; m < nb; m++) {
          key.clear();
          for (int yy = std::max(0, y - 1); yy <= y; yy++)
            for (int xx = 0; xx < Lx; xx++) {
              const int idx = yy * Lx + xx;
              if (idx >= cellidx) break;
              const CellDev& cc = h->cell(yy, xx);
              const unsigned st = hst[(size_t)m * ncell + idx];
              const int a_ = (int)(st & smask), b_ = S == 1 ? a_ : (int)((st >> ns) & smask), cl_ = (int)((st >> (2 * ns)) & hmask);
              if (xx + 1 < Lx && yy * Lx + xx + 1 > cellidx) key.push_back(pext_host(a_, cc.m_right));
              if (yy + 1 < Ly && (yy + 1) * Lx + xx > cellidx) key.push_back(pext_host(b_, cc.m_down));
              if (S == 3 && xx + 1 < Lx && yy + 1 < Ly && (yy + 1) * Lx + xx + 1 > cellidx) key.push_back(pext_host(cl_, cc.m_dout));
            }
          hpid[m] = ids.emplace(key, (int)ids.size()).first->second;
        }
        TN_CUDA(cudaMemcpyAsync(pid.p, hpid.data(), sizeof(int) * nb, cudaMemcpyHostToDevice, h->stream));
        MergeLegs lg{c.Pr, c.Pd, c.Po, c.n_r, c.n_d, c.n_o, x + 1 < Lx, y + 1 < Ly, S == 3 && x + 1 < Lx && y + 1 < Ly};
        int lgA = 0;
        while ((1 << lgA) < c.nA) lgA++;
        const int nchunk = (int)std::max<i64>(1, std::min<i64>(64, per_m / 8192));
        k_sel_fmax<<<cdiv((i64)nb * c.nCl, 256), 256, 0, h->stream>>>(sa, fmx.p, chbest.p);
        TN_LAUNCH_CHECK(h);
        // number of POSSIBLE boundaries of the candidates of this cell
        const double gposs = (double)ids.size() * (lg.use_r ? lg.n_r : 1) * (lg.use_d ? lg.n_d : 1) * (lg.use_o ? lg.n_o : 1);
        const bool seg = h->merge_segmented && gposs <= (double)mcap;
        bool ok = false;
        unsigned n1 = 0, ng = 0;
        int lgClm = 0;
        while ((1 << lgClm) < c.nCl) lgClm++;
        const double mxlp = drops ? d2h(h, scale.p + nb) : 0.0;
        if (seg) {
          // ---- few possible boundaries (always so in the last column and the last row): segmented arg-max over all of V
          const i64 ngroups = (i64)gposs;
          int lgCl = 0;
          while ((1 << lgCl) < c.nCl) lgCl++;
          unsigned long long* gt = gbest.p + mcap;
          unsigned long long* npos = gbest.p + 2 * (size_t)mcap;
          TN_CUDA(cudaMemsetAsync(gbest.p, 0, sizeof(unsigned long long) * ngroups, h->stream));
          TN_CUDA(cudaMemsetAsync(gt, 0xff, sizeof(unsigned long long) * ngroups, h->stream));
          TN_CUDA(cudaMemsetAsync(npos, 0, sizeof(unsigned long long), h->stream));
          TN_CUDA(cudaMemsetAsync(count.p, 0, sizeof(unsigned), h->stream));
          const int nch2 = (int)std::max<i64>(1, std::min<i64>(64, per_m / 4096));
          k_merge_seg<1><<<dim3(nch2, nb), 256, 0, h->stream>>>(sa, lgA, lgCl, fmx.p, chbest.p, pid.p, lg, ns, S, gbest.p, gt, npos);
          TN_LAUNCH_CHECK(h);
          h->st.bytes_search_select += 2.0 * 8.0 * nb * (double)per_m;
          if (!drops) {
            k_merge_seg<2><<<dim3(nch2, nb), 256, 0, h->stream>>>(sa, lgA, lgCl, fmx.p, chbest.p, pid.p, lg, ns, S, gbest.p, gt, npos);
            TN_LAUNCH_CHECK(h);
            k_merge_seg_emit<<<cdiv(ngroups, 256), 256, 0, h->stream>>>(sa, gbest.p, gt, ngroups, lp_cur, Z.p, ns, S, mcands.p, count.p);
            TN_LAUNCH_CHECK(h);
            ng = d2h(h, count.p);
            n1 = (unsigned)std::min<unsigned long long>(d2h(h, npos), 0xffffffffull);
            ok = true;
          } else {
            // droplet mode: every candidate within max_dE of its group's best (all c_hi variants) is needed as a loser
            k_sel_prefilter_all<<<dim3(nch2, nb), 256, 0, h->stream>>>(sa, lgA, lgCl, 0.0, dfac, gbest.p, pid.p, lg, craw.p, count.p, mcap);
            TN_LAUNCH_CHECK(h);
            n1 = d2h(h, count.p);
            if (n1 <= mcap && n1 > 0) {
              n_mc = n1;
              unsigned mp2 = 2;
              while (mp2 < n1 + 1) mp2 <<= 1;
              k_merge_score<<<cdiv(mp2, 256), 256, 0, h->stream>>>(sa, craw.p, n1, mp2, lp_cur, Z.p, ns, S, pid.p, lg, mcand.p);
              TN_LAUNCH_CHECK(h);
              bitonic_sort<MCand, LessM>(h, mcand.p, mp2);
              TN_CUDA(cudaMemsetAsync(count.p, 0, sizeof(unsigned), h->stream));
              k_merge_first<<<cdiv(mp2, 256), 256, 0, h->stream>>>(mcand.p, mp2, mcands.p, count.p);
              TN_LAUNCH_CHECK(h);
              ng = d2h(h, count.p);
              ok = true;
            }
          }
        }
        double thr = 0.0;                                // few candidates: take every positive entry
        if (!seg && !direct) {
          for (int pass = 0; pass < 2; pass++) {
            k_sel_hist<<<gsel, 256, 0, h->stream>>>(sa, sel.p, shifts[pass], nbitsv[pass], pass == 0, 6, hist.p);
            TN_LAUNCH_CHECK(h);
            k_sel_resolve<<<1, 1024, 0, h->stream>>>(sel.p, hist.p, shifts[pass], nbitsv[pass], pass == 0, 0ull);
            TN_LAUNCH_CHECK(h);
          }
          SelState cur = d2h(h, sel.p);
          if (!cur.takeall) {
            long long bits = (long long)cur.thresh;
            memcpy(&thr, &bits, sizeof(double));
            thr *= 1.0 - 1e-12;
          }
        }
        // The threshold is lowered (/ 64) while fewer than M + 1 boundaries lie above it and raised again (geometric
        // bisection) when more candidates than the merge buffers hold lie above it.
        const int max_attempts = 14;   // every attempt is one pass over V
        double thr_few = -1.0, thr_many = -1.0;          // last thresholds with too few groups / too many survivors
        for (int attempt = 0; !seg && attempt < max_attempts; attempt++) {
          TN_CUDA(cudaMemsetAsync(count.p, 0, sizeof(unsigned), h->stream));
          if (drops)
            k_sel_prefilter_all<<<dim3(nchunk, nb), 256, 0, h->stream>>>(sa, lgA, lgClm, thr * dfac, dfac, nullptr, pid.p, lg, craw.p, count.p, mcap);
          else
            k_sel_prefilter_merge<<<dim3(nchunk, nb), 256, 0, h->stream>>>(sa, lgA, thr, fmx.p, craw.p, count.p, mcap);
          h->st.bytes_search_select += 8.0 * nb * (double)per_m * (attempt == 0 && !direct ? 1.0 + 2.0 / 64.0 : 1.0);
          TN_LAUNCH_CHECK(h);
          n1 = d2h(h, count.p);
          if (n1 > mcap) {                               // too many survivors for the merge buffers
            if (thr <= 0.0) {                                                   // every positive entry, still too many:
              if (thr_few <= 0.0) break;                                        //   nothing to bisect against
              thr_many = thr_few * 1e-80;                                       //   the bound lies somewhere below thr_few
            } else {
              thr_many = thr;
            }
            if (thr_few > 0.0 && !(thr_few > thr_many * (1.0 + 1e-9))) break;   // the two bounds met: no threshold fits
            thr = thr_few > 0.0 ? std::sqrt(thr_few) * std::sqrt(thr_many) : thr * 8.0;
            continue;
          }
          if (n1 == 0 && thr == 0.0) break;
          unsigned mp2 = 2;
          while (mp2 < n1 + 1) mp2 <<= 1;
          k_merge_score<<<cdiv(mp2, 256), 256, 0, h->stream>>>(sa, craw.p, n1, mp2, lp_cur, Z.p, ns, S, pid.p, lg, mcand.p);
          TN_LAUNCH_CHECK(h);
          bitonic_sort<MCand, LessM>(h, mcand.p, mp2);
          TN_CUDA(cudaMemsetAsync(count.p, 0, 2 * sizeof(unsigned), h->stream));
          k_merge_first<<<cdiv(mp2, 256), 256, 0, h->stream>>>(mcand.p, mp2, mcands.p, count.p,
                                                               drops && thr > 0.0 ? std::log(thr) + mxlp : -INFINITY,
                                                               drops ? count.p + 1 : nullptr);
          TN_LAUNCH_CHECK(h);
          ng = d2h(h, count.p);
          n_mc = n1;
          // droplet mode: the list reaches down to thr * dfac, but M + 1 WINNERS must lie at or above thr itself
          const unsigned ng_sel = drops ? d2h(h, count.p + 1) : ng;
          if (ng_sel >= (unsigned)M + 1 || thr == 0.0) { ok = true; break; }
          thr_few = thr;                                 // fewer than M + 1 boundaries above the bound: lower it
          if (thr_many > 0.0) thr = std::sqrt(thr_few) * std::sqrt(thr_many);
          else thr = (attempt < 3 && thr > 1e-290) ? thr / 64.0 : 0.0;       // a few steps down, then every positive entry
        }
        if (ok) {
          if (ng == 0) tn_throw(TN_ERR_NUMERIC, "cell (%d,%d): every candidate has zero probability", y, x);
          h->st.merged_away += (int64_t)n1 - (int64_t)ng;
          while (np2 < ng + 1) np2 <<= 1;
          while (np2 <= (unsigned)M) np2 <<= 1;
          k_fill_sentinel<<<cdiv(np2 - ng, 256), 256, 0, h->stream>>>(mcands.p, ng, np2);
          TN_LAUNCH_CHECK(h);
          bitonic_sort<Cand, LessC>(h, mcands.p, np2);
          ncand = ng;
          cand_sorted = true;
        } else {
          // more survivors than the merge buffers hold at every threshold tried: this cell is selected WITHOUT merging
          // (counted: a run with merge_fallback_cells > 0 is not the algorithm of Fig. 3(d) at those cells)
          h->st.merge_fallback_cells++;
          TN_CUDA(cudaMemcpyAsync(sel.p, &s0, sizeof(s0), cudaMemcpyHostToDevice, h->stream));
          TN_CUDA(cudaMemsetAsync(hist.p, 0, sizeof(unsigned) * 4096, h->stream));
        }
      }
      if (cand_sorted) {
        // nothing: the merged route produced the sorted candidate list
      } else if (!direct) {
        k_sel_fmax<<<cdiv((i64)nb * c.nCl, 256), 256, 0, h->stream>>>(sa, fmx.p);
        TN_LAUNCH_CHECK(h);
        // (1) lower bound of the (M+1)-th largest key from a SUBSET of the candidates (two radix digits): the row maxima
        //     that k_cond wrote (one candidate per row of V), else a hashed 1/64 sample of V
        for (int pass = 0; pass < 2; pass++) {
          if (have_rowmax) {
            const int Mg = c.nB * c.nCl;
            k_sel_hist_rows<<<(unsigned)std::min<i64>((i64)h->sms * 8, ((i64)nb * Mg + 255) / 256), 256, 0, h->stream>>>(
                rowmax.p, scale.p, fmx.p, nb, Mg, c.nCl, sel.p, shifts[pass], nbitsv[pass], pass == 0, hist.p);
          } else {
            k_sel_hist<<<gsel, 256, 0, h->stream>>>(sa, sel.p, shifts[pass], nbitsv[pass], pass == 0, 6, hist.p);
          }
          TN_LAUNCH_CHECK(h);
          k_sel_resolve<<<1, 1024, 0, h->stream>>>(sel.p, hist.p, shifts[pass], nbitsv[pass], pass == 0, 0ull);
          TN_LAUNCH_CHECK(h);
        }
        // lazy V: the rows that reach the bound are computed now (the others are never written, never read)
        if (lazy_v) launch_cond_rows(h, nb, ca_rows, sel.p, scale.p, fmx.p);
        // (2) one pass over V (only the rows whose maximum reaches the bound are read when the row maxima are there):
        //     everything at or above the bound goes to the compact list
        TN_CUDA(cudaMemsetAsync(count.p, 0, sizeof(unsigned), h->stream));
        {
          int lgA = 0;
          while ((1 << lgA) < c.nA) lgA++;
          const int nchunk = (int)std::max<i64>(1, std::min<i64>(64, per_m / 8192));
          k_sel_prefilter<<<dim3(nchunk, nb), 256, 0, h->stream>>>(sa, lgA, sel.p, fmx.p, ckeys.p, craw.p, count.p, ccap,
                                                                   have_rowmax ? rowmax.p : nullptr);
          // algorithmic bytes: with the row maxima 8 B per row (three times) instead of one read of V + the sample
          h->st.bytes_search_select += have_rowmax ? 3.0 * 8.0 * nb * (double)c.nB * c.nCl
                                                   : 8.0 * nb * (double)per_m * (1.0 + 2.0 / 64.0);
        }
        TN_LAUNCH_CHECK(h);
        const unsigned n1 = d2h(h, count.p);
        if (n1 > ccap) {
          direct = true;                              // massive ties at the bound: fall back to the direct passes
          if (lazy_v) {                               // ... which read all of V: write it now (no second tally of Z)
            ca_rows.store = 1;
            ca_rows.tally = 0;
            if (!launch_cond(h, nb, ca_rows)) tn_throw(TN_ERR_CUDA, "cell (%d,%d): lazy V could not be completed", y, x);
            lazy_v = false;
          }
        } else if (n1 <= cap) {
          ncand = n1;
          TN_CUDA(cudaMemcpyAsync(raw.p, craw.p, sizeof(Raw) * n1, cudaMemcpyDeviceToDevice, h->stream));
        } else {
          // (3) exact radix selection on the compact keys
          TN_CUDA(cudaMemcpyAsync(sel.p, &s0, sizeof(s0), cudaMemcpyHostToDevice, h->stream));
          const int gc = (int)std::min<i64>((i64)h->sms * 4, ((i64)n1 + 255) / 256);
          for (int pass = 0; pass < 6; pass++) {
            k_csel_hist<<<gc, 256, 0, h->stream>>>(ckeys.p, n1, sel.p, shifts[pass], nbitsv[pass], pass == 0, hist.p);
            TN_LAUNCH_CHECK(h);
            k_sel_resolve<<<1, 1024, 0, h->stream>>>(sel.p, hist.p, shifts[pass], nbitsv[pass], pass == 0, cap);
            TN_LAUNCH_CHECK(h);
            SelState cur = d2h(h, sel.p);
            if (cur.done) break;
          }
          TN_CUDA(cudaMemsetAsync(count.p, 0, sizeof(unsigned), h->stream));
          k_csel_compact<<<gc, 256, 0, h->stream>>>(ckeys.p, craw.p, n1, sel.p, raw.p, count.p, cap);
          TN_LAUNCH_CHECK(h);
          ncand = d2h(h, count.p);
          if (ncand > cap) {   // more ties at the cut than the list holds: collect ALL of them (deterministic, S8 order)
            if (ncand <= tie_cap) {
              rawL.reset(new DBuf<Raw>(h, ncand));
              TN_CUDA(cudaMemsetAsync(count.p, 0, sizeof(unsigned), h->stream));
              k_csel_compact<<<gc, 256, 0, h->stream>>>(ckeys.p, craw.p, n1, sel.p, rawL->p, count.p, ncand);
              TN_LAUNCH_CHECK(h);
              h->st.select_tie_overflow++;
            } else {
              h->st.select_tie_dropped++;
              ncand = cap;
            }
          }
        }
      }
      if (direct && !cand_sorted) {
        TN_CUDA(cudaMemcpyAsync(sel.p, &s0, sizeof(s0), cudaMemcpyHostToDevice, h->stream));
        TN_CUDA(cudaMemsetAsync(hist.p, 0, sizeof(unsigned) * 4096, h->stream));
        for (int pass = 0; pass < 6; pass++) {
          k_sel_hist<<<gsel, 256, 0, h->stream>>>(sa, sel.p, shifts[pass], nbitsv[pass], pass == 0, 0, hist.p);
          TN_LAUNCH_CHECK(h);
          k_sel_resolve<<<1, 1024, 0, h->stream>>>(sel.p, hist.p, shifts[pass], nbitsv[pass], pass == 0, cap);
          TN_LAUNCH_CHECK(h);
          SelState cur = d2h(h, sel.p);
          if (cur.done) break;
        }
        TN_CUDA(cudaMemsetAsync(count.p, 0, sizeof(unsigned), h->stream));
        k_sel_collect<<<gsel, 256, 0, h->stream>>>(sa, sel.p, raw.p, count.p, cap);
        TN_LAUNCH_CHECK(h);
        ncand = d2h(h, count.p);
        if (ncand > cap) {     // more ties at the cut than the list holds: collect ALL of them (deterministic, S8 order)
          if (ncand <= tie_cap) {
            rawL.reset(new DBuf<Raw>(h, ncand));
            TN_CUDA(cudaMemsetAsync(count.p, 0, sizeof(unsigned), h->stream));
            k_sel_collect<<<gsel, 256, 0, h->stream>>>(sa, sel.p, rawL->p, count.p, ncand);
            TN_LAUNCH_CHECK(h);
            h->st.select_tie_overflow++;
          } else {
            h->st.select_tie_dropped++;
            ncand = cap;
          }
        }
      }
      if (ncand == 0) tn_throw(TN_ERR_NUMERIC, "cell (%d,%d): every candidate has zero probability", y, x);
      Cand* cand_final = cand_sorted ? mcands.p : cand.p;
      if (!cand_sorted) {
      while (np2 < ncand + 1) np2 <<= 1;   // at least one sentinel so that cand[M] exists when ncand <= M
      while (np2 <= (unsigned)M) np2 <<= 1;
      if (rawL) {                          // tie overflow: the complete tie group, in buffers of its own
        candL.reset(new DBuf<Cand>(h, np2));
        cand_final = candL->p;
      } else if (np2 > npad) {
        np2 = npad;
      }
      k_sel_score<<<cdiv(np2, 256), 256, 0, h->stream>>>(sa, rawL ? rawL->p : raw.p, ncand, np2, lp_cur, Z.p, ns, S, cand_final);
      TN_LAUNCH_CHECK(h);
      if (np2 <= 4096) {
        k_bitonic_smem<<<1, 1024, np2 * sizeof(Cand), h->stream>>>(cand_final, np2);
        TN_LAUNCH_CHECK(h);
      } else {
        bitonic_sort<Cand, LessC>(h, cand_final, np2);   // tiled: a handful of launches instead of log^2 n
      }
      }
      const int nkeep = (int)std::min<unsigned>(ncand, (unsigned)M);
      k_new_beam<<<nkeep, 128, 0, h->stream>>>(cand_final, nkeep, M, st_cur, st_nxt, ncell, cellidx, sl_cur, sl_nxt, lp_nxt,
                                               LG.p, npp, Dr, ldLv, Lv_nxt, c.Pd, c.Po, c.n_o, ns, S, pd.p);
      TN_LAUNCH_CHECK(h);
      if (drops) {
        if (cand_sorted && n_mc > 0) {
          MergeLegs lgd{c.Pr, c.Pd, c.Po, c.n_r, c.n_d, c.n_o, x + 1 < Lx, y + 1 < Ly, S == 3 && x + 1 < Lx && y + 1 < Ly};
          DropArgs da{mcand.p, n_mc, cand_final, nkeep, st_cur, ncell, cellidx, pid.p, lgd, ns, S, c.nCl,
                      dp_cur, dd_cur, dc_cur, dp_nxt, dd_nxt, dc_nxt, dK, h->droplet_max_dE, h->beta, h->droplet_min_hamming,
                      d_spin_of.p, nbits, d_adj_ptr.p, d_adj.p, h->n_spins, d_dover.p};
          k_droplets<<<nkeep, 128, drop_smem, h->stream>>>(da);
          TN_LAUNCH_CHECK(h);
        } else {
          k_droplets_inherit<<<nkeep, 128, 0, h->stream>>>(cand_final, nkeep, dK, ncell, dp_cur, dd_cur, dc_cur, dp_nxt, dd_nxt, dc_nxt);
          TN_LAUNCH_CHECK(h);
        }
        std::swap(dp_cur, dp_nxt); std::swap(dd_cur, dd_nxt); std::swap(dc_cur, dc_nxt);
      }
      std::swap(st_cur, st_nxt); std::swap(lp_cur, lp_nxt); std::swap(Lv_cur, Lv_nxt); std::swap(sl_cur, sl_nxt);
      nb = nkeep;
      t_s.stop();
    }
    for (auto& r : rt) { h->dfree(r.G); h->dfree(r.RM); h->dfree(r.ls); }
  }
  // ---- outputs: logp is already sorted descending (selection order)
  DBuf<int8_t> sp(h, (size_t)nb * h->n_spins);
  DBuf<double> E(h, nb);
  k_unpack<<<cdiv((i64)nb * h->n_spins, 256), 256, 0, h->stream>>>(st_cur, ncell, nb, h->n_spins, h->d_cell_of, h->d_bit_of, sp.p);
  TN_LAUNCH_CHECK(h);
  k_energy<<<cdiv(nb, 64), 64, 0, h->stream>>>(sp.p, nb, h->n_spins, h->n_edges, h->d_eu, h->d_ev, h->d_J, h->d_h, E.p);
  TN_LAUNCH_CHECK(h);
  TN_CUDA(cudaMemcpyAsync(states_out, sp.p, (size_t)nb * h->n_spins, cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaMemcpyAsync(energies, E.p, sizeof(double) * nb, cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaMemcpyAsync(logp_out, lp_cur, sizeof(double) * nb, cudaMemcpyDeviceToHost, h->stream));
  double pdv = 0;
  TN_CUDA(cudaMemcpyAsync(&pdv, pd.p, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  unsigned long long neg = 0;
  TN_CUDA(cudaMemcpyAsync(&neg, nneg.p, sizeof(neg), cudaMemcpyDeviceToHost, h->stream));
  h->drop_cnt.clear(); h->drop_dE.clear(); h->drop_flips.clear();
  h->drop_K = 0;
  if (drops) {
    DBuf<int8_t> dfl(h, (size_t)nb * dK * h->n_spins);
    k_droplets_unpack<<<cdiv((i64)nb * dK * h->n_spins, 256), 256, 0, h->stream>>>(dp_cur, nb, dK, ncell, h->n_spins, h->d_cell_of,
                                                                                  h->d_bit_of, dfl.p);
    TN_LAUNCH_CHECK(h);
    h->drop_K = dK;
    h->drop_cnt.resize(nb); h->drop_dE.resize((size_t)nb * dK); h->drop_flips.resize((size_t)nb * dK * h->n_spins);
    TN_CUDA(cudaMemcpyAsync(h->drop_cnt.data(), dc_cur, sizeof(int) * nb, cudaMemcpyDeviceToHost, h->stream));
    TN_CUDA(cudaMemcpyAsync(h->drop_dE.data(), dd_cur, sizeof(double) * nb * dK, cudaMemcpyDeviceToHost, h->stream));
    TN_CUDA(cudaMemcpyAsync(h->drop_flips.data(), dfl.p, (size_t)nb * dK * h->n_spins, cudaMemcpyDeviceToHost, h->stream));
    unsigned long long over = 0;
    TN_CUDA(cudaMemcpyAsync(&over, d_dover.p, sizeof(over), cudaMemcpyDeviceToHost, h->stream));
    TN_CUDA(cudaStreamSynchronize(h->stream));
    h->st.droplet_overflow += (int64_t)over;
  }
  TN_CUDA(cudaStreamSynchronize(h->stream));
  *n_out = nb;
  if (log_pd_out) *log_pd_out = pdv;
  h->st.negative_u += (int64_t)neg;
}

}  // namespace

void search_logz(tn_handle* h) { run(h, 1, true, nullptr, nullptr, nullptr, nullptr, nullptr); }

void search_run(tn_handle* h, int M, int* n_out, int8_t* states, double* energies, double* logp, double* log_pd) {
  cudaEvent_t e0, e1;
  TN_CUDA(cudaEventCreate(&e0)); TN_CUDA(cudaEventCreate(&e1));
  TN_CUDA(cudaEventRecord(e0, h->stream));
  try {
    run(h, M, false, n_out, states, energies, logp, log_pd);
  } catch (...) {
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    throw;
  }
  TN_CUDA(cudaEventRecord(e1, h->stream));
  TN_CUDA(cudaEventSynchronize(e1));
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  h->st.ms_search += ms;
}

void energy_run(tn_handle* h, int n, const int8_t* states, double* energies) {
  if (n == 0) return;
  DBuf<int8_t> sp(h, (size_t)n * h->n_spins);
  DBuf<double> E(h, n);
  TN_CUDA(cudaMemcpyAsync(sp.p, states, (size_t)n * h->n_spins, cudaMemcpyHostToDevice, h->stream));
  k_energy<<<cdiv(n, 64), 64, 0, h->stream>>>(sp.p, n, h->n_spins, h->n_edges, h->d_eu, h->d_ev, h->d_J, h->d_h, E.p);
  TN_LAUNCH_CHECK(h);
  TN_CUDA(cudaMemcpyAsync(energies, E.p, sizeof(double) * n, cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaStreamSynchronize(h->stream));
}
