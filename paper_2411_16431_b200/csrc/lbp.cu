// f4: local dimensional reduction by loopy belief propagation (Sec. IV, Eqs. (11)-(13), Fig. 9).
//
// Messages live on the directed neighbour pairs of the cell grid; legs of a cell: 0 left, 1 right, 2 up, 3 down,
// 4 din, 5 dout.  nu[cell][leg][.] = message arriving over that leg (a vector over the leg's projected index, Eq. (5)),
// mu[cell][leg][.] = message the cell sends towards that leg's edge; mu[cell][6][0] = the cell's normaliser of Eq. (13).
//   Eq. (11)  mu_leg(xbar) = sum_{x : P_leg(x) = xbar} w(x) prod_{leg' != leg} nu_leg'(P_leg'(x))
//   Eq. (12)  nu_leg(xbar_n) = sum_{xbar_m} exp(-beta Ebar)[xbar_m, xbar_n] mu^{neighbour}_{opposite leg}(xbar_m)
//   Eq. (13)  p(x) ~ w(x) prod_leg nu_leg(P_leg(x))
// The paper sums Eq. (11) over all d cell states with the projectors keeping the messages small.  Here the
// cell weight is the chain  w = wA[a] X[a_hi][b] Yc[b][c_lo] wC[c_lo][c_hi]  (tn_common.cuh), so the sum over 2^24 states
// is a chain of four small contractions (256 x 256 at most), one CTA per (cell, leg), every reduction in a fixed order.
// Readings: DESIGN.md S26 (uniform start, all mu then all nu per iteration, nu normalised to sum 1, absent or uncoupled
// neighbours send the constant 1, top-K order = p descending then state ascending).
#include "kernels.cuh"
#include <algorithm>

namespace {

constexpr int LBP_LD = 256;   // leg ranges are <= 256

struct LbpShared {
  double gA[256], gB[256], yB[256], hB[256], hT[256], kA[256], mB[256];
  double gCl[16], gCh[16], sC[16], hC[16], nC[16];
};

// factors of cell c with the incoming message of leg `skip` replaced by 1 (skip = 6: none)
__device__ void lbp_factors(const CellDev& c, const double* nu_cell, int skip, LbpShared& s) {
  const int tid = threadIdx.x;
  const double* nL = nu_cell + 0 * LBP_LD;
  const double* nR = nu_cell + 1 * LBP_LD;
  const double* nU = nu_cell + 2 * LBP_LD;
  const double* nD = nu_cell + 3 * LBP_LD;
  const double* nI = nu_cell + 4 * LBP_LD;
  const double* nO = nu_cell + 5 * LBP_LD;
  for (int a = tid; a < c.nA; a += blockDim.x)
    s.gA[a] = c.wA[a] * (skip == 0 ? 1.0 : nL[c.Pl[a]]) * (skip == 1 ? 1.0 : nR[c.Pr[a]]);
  for (int b = tid; b < c.nB; b += blockDim.x) s.gB[b] = (skip == 2 ? 1.0 : nU[c.Pu[b]]) * (skip == 3 ? 1.0 : nD[c.Pd[b]]);
  if (tid < c.nCh) s.gCh[tid] = skip == 4 ? 1.0 : nI[c.Pi[tid]];
  if (tid < c.nCl) s.gCl[tid] = skip == 5 ? 1.0 : nO[c.Po[tid]];
  __syncthreads();
  if (tid < c.nCl) {
    double t = 0.0;
    for (int ch = 0; ch < c.nCh; ch++) t += c.wC[tid * c.nCh + ch] * s.gCh[ch];
    s.sC[tid] = t;
    s.hC[tid] = s.gCl[tid] * t;
  }
  __syncthreads();
  for (int b = tid; b < c.nB; b += blockDim.x) {
    double t = 0.0;
    for (int cl = 0; cl < c.nCl; cl++) t += c.Yc[b * c.nCl + cl] * s.hC[cl];
    s.yB[b] = t;
    s.hB[b] = s.gB[b] * t;
  }
  __syncthreads();
  for (int t = tid; t < c.nT; t += blockDim.x) {
    double acc = 0.0, ka = 0.0;
    for (int b = 0; b < c.nB; b++) acc += c.X[t * c.nB + b] * s.hB[b];
    s.hT[t] = acc;
    for (int a = 0; a < c.nA; a++)
      if ((a >> c.tshift) == t) ka += s.gA[a];
    s.kA[t] = ka;
  }
  __syncthreads();
  for (int b = tid; b < c.nB; b += blockDim.x) {
    double acc = 0.0;
    for (int t = 0; t < c.nT; t++) acc += s.kA[t] * c.X[t * c.nB + b];
    s.mB[b] = acc;
  }
  __syncthreads();
  if (tid < c.nCl) {
    double acc = 0.0;
    for (int b = 0; b < c.nB; b++) acc += s.gB[b] * s.mB[b] * c.Yc[b * c.nCl + tid];
    s.nC[tid] = acc;
  }
  __syncthreads();
}

// Eq. (11): grid (cell, 7); leg 6 = the normaliser of Eq. (13)
__global__ void __launch_bounds__(256) k_lbp_mu(const CellDev* cells, const double* nu, double* mu) {
  __shared__ LbpShared s;
  const int cell = blockIdx.x, leg = blockIdx.y, tid = threadIdx.x;
  const CellDev c = cells[cell];
  lbp_factors(c, nu + (size_t)cell * 6 * LBP_LD, leg, s);
  double* out = mu + ((size_t)cell * 7 + leg) * LBP_LD;
  if (leg == 0 || leg == 1) {
    const int n = leg == 0 ? c.n_l : c.n_r;
    const int* P = leg == 0 ? c.Pl : c.Pr;
    if (tid < n) {
      double acc = 0.0;
      for (int a = 0; a < c.nA; a++)
        if (P[a] == tid) acc += s.gA[a] * s.hT[a >> c.tshift];
      out[tid] = acc;
    }
  } else if (leg == 2 || leg == 3) {
    const int n = leg == 2 ? c.n_u : c.n_d;
    const int* P = leg == 2 ? c.Pu : c.Pd;
    if (tid < n) {
      double acc = 0.0;
      for (int b = 0; b < c.nB; b++)
        if (P[b] == tid) acc += s.gB[b] * s.mB[b] * s.yB[b];
      out[tid] = acc;
    }
  } else if (leg == 5) {
    if (tid < c.n_o) {
      double acc = 0.0;
      for (int cl = 0; cl < c.nCl; cl++)
        if (c.Po[cl] == tid) acc += s.nC[cl] * s.sC[cl];
      out[tid] = acc;
    }
  } else if (leg == 4) {
    if (tid < c.n_i) {
      double acc = 0.0;
      for (int ch = 0; ch < c.nCh; ch++)
        if (c.Pi[ch] == tid) {
          double t = 0.0;
          for (int cl = 0; cl < c.nCl; cl++) t += c.wC[cl * c.nCh + ch] * s.gCl[cl] * s.nC[cl];
          acc += t;
        }
      out[tid] = acc;
    }
  } else if (tid == 0) {
    double acc = 0.0;
    for (int a = 0; a < c.nA; a++) acc += s.gA[a] * s.hT[a >> c.tshift];
    out[0] = acc;
  }
}

// Eq. (12) + normalisation: grid (cell, 6)
__global__ void __launch_bounds__(256) k_lbp_nu(const CellDev* cells, const double* mu, double* nu, int Ly, int Lx, int S) {
  __shared__ double v[256];
  __shared__ double s_sum;
  const int cell = blockIdx.x, leg = blockIdx.y, tid = threadIdx.x;
  const int y = cell / Lx, x = cell % Lx;
  const CellDev c = cells[cell];
  const int dy[6] = {0, 0, -1, 1, -1, 1}, dx[6] = {-1, 1, 0, 0, -1, 1}, back[6] = {1, 0, 3, 2, 5, 4};
  const int n = leg == 0 ? c.n_l : leg == 1 ? c.n_r : leg == 2 ? c.n_u : leg == 3 ? c.n_d : leg == 4 ? c.n_i : c.n_o;
  const int yy = y + dy[leg], xx = x + dx[leg];
  const bool exists = yy >= 0 && yy < Ly && xx >= 0 && xx < Lx && (leg < 4 || S == 3);
  double* out = nu + ((size_t)cell * 6 + leg) * LBP_LD;
  if (!exists) {
    if (tid < n) out[tid] = 1.0;
    return;
  }
  const int ncell = yy * Lx + xx;
  const CellDev cn = cells[ncell];
  const double* m = mu + ((size_t)ncell * 7 + back[leg]) * LBP_LD;
  if (tid < n) {
    double acc = 0.0;
    if (leg == 0) for (int r = 0; r < c.bh_rows; r++) acc += c.Bh[r * c.n_l + tid] * m[r];
    else if (leg == 1) for (int l = 0; l < cn.n_l; l++) acc += cn.Bh[tid * cn.n_l + l] * m[l];
    else if (leg == 2) for (int p = 0; p < c.bv_rows; p++) acc += c.Bv[p * c.n_u + tid] * m[p];
    else if (leg == 3) for (int u = 0; u < cn.n_u; u++) acc += cn.Bv[tid * cn.n_u + u] * m[u];
    else if (leg == 4) for (int q = 0; q < c.bd_rows; q++) acc += c.Bd[q * c.n_i + tid] * m[q];
    else for (int i = 0; i < cn.n_i; i++) acc += cn.Bd[tid * cn.n_i + i] * m[i];
    v[tid] = acc;
  }
  __syncthreads();
  if (tid == 0) {
    double t = 0.0;
    for (int i = 0; i < n; i++) t += v[i];
    s_sum = t;
  }
  __syncthreads();
  if (tid < n) out[tid] = v[tid] / s_sum;
}

__device__ __forceinline__ double lbp_weight(const CellDev& c, const LbpShared& s, unsigned st, int ns, int S) {
  const unsigned smask = (1u << ns) - 1, hmask = (1u << (ns / 2)) - 1;
  const int a = (int)(st & smask), b = S == 1 ? a : (int)((st >> ns) & smask);
  const int cl = S == 3 ? (int)((st >> (2 * ns)) & hmask) : 0, ch = S == 3 ? (int)((st >> (2 * ns + ns / 2)) & hmask) : 0;
  return s.gA[a] * c.X[(a >> c.tshift) * c.nB + b] * s.gB[b] * c.Yc[b * c.nCl + cl] * s.gCl[cl] * c.wC[cl * c.nCh + ch] * s.gCh[ch];
}
// Eq. (13) at given states (log of the normalised marginal), or for ALL states when `states` is NULL (p itself, not log)
__global__ void __launch_bounds__(256) k_lbp_eval(const CellDev* cells, int cell, const double* nu, const double* mu, int ns, int S,
                                                  i64 n, const unsigned* states, double* out) {
  __shared__ LbpShared s;
  const CellDev c = cells[cell];
  lbp_factors(c, nu + (size_t)cell * 6 * LBP_LD, 6, s);
  const double Z = mu[((size_t)cell * 7 + 6) * LBP_LD];
  for (i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (i64)gridDim.x * blockDim.x) {
    const unsigned st = states ? states[t] : (unsigned)t;
    const double w = lbp_weight(c, s, st, ns, S);
    out[t] = states ? log(w / Z) : w / Z;
  }
}

// ---- top-K of a positive array: radix histogram on the key bits (host-resolved, 12 bits per pass), compaction, sort
struct PS { double p; unsigned st; unsigned pad; };
__global__ void k_lbp_hist(const double* p, i64 n, int shift, unsigned long long prefix, int first, unsigned* hist) {
  __shared__ unsigned sh[4096];
  for (int i = threadIdx.x; i < 4096; i += blockDim.x) sh[i] = 0;
  __syncthreads();
  for (i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (i64)gridDim.x * blockDim.x) {
    const unsigned long long key = (unsigned long long)__double_as_longlong(p[t]);
    if (!first && (key >> (shift + 12)) != prefix) continue;
    atomicAdd(&sh[(key >> shift) & 4095u], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 4096; i += blockDim.x)
    if (sh[i]) atomicAdd(&hist[i], sh[i]);
}
__global__ void k_lbp_collect(const double* p, i64 n, double thr, PS* out, unsigned* count, unsigned cap) {
  for (i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (i64)gridDim.x * blockDim.x)
    if (p[t] >= thr) {
      const unsigned idx = atomicAdd(count, 1u);
      if (idx < cap) out[idx] = PS{p[t], (unsigned)t, 0u};
    }
}
__global__ void k_lbp_pad(PS* c, unsigned from, unsigned to) {
  const unsigned t = from + blockIdx.x * blockDim.x + threadIdx.x;
  if (t < to) c[t] = PS{-1.0, 0xffffffffu, 0u};
}
__global__ void k_lbp_bitonic(PS* c, unsigned n, unsigned k, unsigned j) {
  const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const unsigned l = i ^ j;
  if (l > i) {
    const PS x = c[i], y = c[l];
    const bool xy = x.p > y.p || (x.p == y.p && x.st < y.st);   // x before y: p descending, state ascending
    const bool up = (i & k) == 0;
    if (up ? !xy : xy) { c[i] = y; c[l] = x; }
  }
}

void need_lbp(tn_handle* h, int y, int x) {
  if (!h->have_lbp) tn_throw(TN_ERR_STATE, "tn_lbp has not run since the last tn_set_beta");
  if (y < 0 || y >= h->Ly || x < 0 || x >= h->Lx) tn_throw(TN_ERR_ARG, "cell (%d, %d) out of range", y, x);
}

}  // namespace

void lbp_free(tn_handle* h) {
  if (h->lbp_nu) h->dfree(h->lbp_nu);
  if (h->lbp_mu) h->dfree(h->lbp_mu);
  h->lbp_nu = h->lbp_mu = nullptr;
  h->have_lbp = false;
}

void lbp_run(tn_handle* h, int iterations) {
  const int ncell = h->Ly * h->Lx;
  if (!h->lbp_nu) h->lbp_nu = h->dalloc<double>((size_t)ncell * 6 * LBP_LD);
  if (!h->lbp_mu) h->lbp_mu = h->dalloc<double>((size_t)ncell * 7 * LBP_LD);
  fill_value(h, h->lbp_nu, (i64)ncell * 6 * LBP_LD, 1.0);                  // uniform start
  for (int it = 0; it < iterations; it++) {
    k_lbp_mu<<<dim3(ncell, 6), 256, 0, h->stream>>>(h->d_cells, h->lbp_nu, h->lbp_mu);      // Fig. 9(c)
    TN_LAUNCH_CHECK(h);
    k_lbp_nu<<<dim3(ncell, 6), 256, 0, h->stream>>>(h->d_cells, h->lbp_mu, h->lbp_nu, h->Ly, h->Lx, h->S);   // Fig. 9(d)
    TN_LAUNCH_CHECK(h);
  }
  k_lbp_mu<<<dim3(ncell, 7), 256, 0, h->stream>>>(h->d_cells, h->lbp_nu, h->lbp_mu);        // normalisers of Eq. (13)
  TN_LAUNCH_CHECK(h);
  TN_CUDA(cudaStreamSynchronize(h->stream));
  h->have_lbp = true;
}

void lbp_message(tn_handle* h, int y, int x, int leg, int* n, double* out) {
  need_lbp(h, y, x);
  if (leg < 0 || leg > 5) tn_throw(TN_ERR_ARG, "leg must be 0..5");
  const CellDev& c = h->cell(y, x);
  const int sz[6] = {c.n_l, c.n_r, c.n_u, c.n_d, c.n_i, c.n_o};
  *n = sz[leg];
  TN_CUDA(cudaMemcpyAsync(out, h->lbp_nu + ((size_t)(y * h->Lx + x) * 6 + leg) * LBP_LD, sizeof(double) * sz[leg],
                          cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaStreamSynchronize(h->stream));
}

void lbp_marginals(tn_handle* h, int y, int x, i64 n, const unsigned* states, double* logp) {
  need_lbp(h, y, x);
  if (n <= 0) return;
  const int nbits = h->S * h->ns;
  for (i64 i = 0; i < n; i++)
    if (nbits < 32 && (states[i] >> nbits)) tn_throw(TN_ERR_ARG, "cell state %u has bits beyond the cell's %d spins", states[i], nbits);
  DBuf<unsigned> ds(h, (size_t)n);
  DBuf<double> dl(h, (size_t)n);
  TN_CUDA(cudaMemcpyAsync(ds.p, states, sizeof(unsigned) * n, cudaMemcpyHostToDevice, h->stream));
  k_lbp_eval<<<(unsigned)std::min<i64>(1024, (n + 255) / 256), 256, 0, h->stream>>>(h->d_cells, y * h->Lx + x, h->lbp_nu, h->lbp_mu,
                                                                                  h->ns, h->S, n, ds.p, dl.p);
  TN_LAUNCH_CHECK(h);
  TN_CUDA(cudaMemcpyAsync(logp, dl.p, sizeof(double) * n, cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaStreamSynchronize(h->stream));
}

void lbp_select(tn_handle* h, int y, int x, int K, int* n_out, unsigned* states, double* logp) {
  need_lbp(h, y, x);
  const int nbits = h->S * h->ns;
  const i64 d = (i64)1 << nbits;
  if (K < 1 || K > (1 << 20)) tn_throw(TN_ERR_ARG, "K must be in 1..2^20");
  const i64 Keff = std::min<i64>(K, d);
  DBuf<double> p(h, (size_t)d);
  const unsigned grid = (unsigned)std::min<i64>((i64)h->sms * 8, (d + 255) / 256);
  k_lbp_eval<<<grid, 256, 0, h->stream>>>(h->d_cells, y * h->Lx + x, h->lbp_nu, h->lbp_mu, h->ns, h->S, d, nullptr, p.p);
  TN_LAUNCH_CHECK(h);
  // threshold = lower edge of the radix bin that holds the Keff-th largest key (positive doubles order like integers)
  DBuf<unsigned> hist(h, 4096), count(h, 1);
  std::vector<unsigned> hh(4096);
  unsigned long long prefix = 0;
  i64 want = Keff;
  int shift = 52;
  for (int pass = 0; pass < 4; pass++) {
    shift = 52 - 12 * pass;
    TN_CUDA(cudaMemsetAsync(hist.p, 0, sizeof(unsigned) * 4096, h->stream));
    k_lbp_hist<<<grid, 256, 0, h->stream>>>(p.p, d, shift, prefix, pass == 0, hist.p);
    TN_LAUNCH_CHECK(h);
    TN_CUDA(cudaMemcpyAsync(hh.data(), hist.p, sizeof(unsigned) * 4096, cudaMemcpyDeviceToHost, h->stream));
    TN_CUDA(cudaStreamSynchronize(h->stream));
    int bin = 4095;
    i64 above = 0;
    for (; bin > 0; bin--) {
      if (above + hh[bin] >= want) break;
      above += hh[bin];
    }
    want -= above;
    prefix = pass == 0 ? (unsigned long long)bin : ((prefix << 12) | (unsigned long long)bin);
    if ((i64)hh[bin] <= 65536) break;          // the bin's members all fit the candidate list
  }
  unsigned long long tbits = prefix << shift;
  double thr;
  memcpy(&thr, &tbits, sizeof(double));
  unsigned cap = (unsigned)Keff + 65536u + 4096u, np2 = 2;
  while (np2 < cap) np2 <<= 1;
  DBuf<PS> cand(h, np2);
  TN_CUDA(cudaMemsetAsync(count.p, 0, sizeof(unsigned), h->stream));
  k_lbp_collect<<<grid, 256, 0, h->stream>>>(p.p, d, thr, cand.p, count.p, np2);
  TN_LAUNCH_CHECK(h);
  unsigned got = 0;
  TN_CUDA(cudaMemcpyAsync(&got, count.p, sizeof(unsigned), cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaStreamSynchronize(h->stream));
  if (got > np2) tn_throw(TN_ERR_NUMERIC, "tn_lbp_select: %u states tie at the cut (more than the list of %u holds)", got, np2);
  if (got < np2) {
    k_lbp_pad<<<cdiv(np2 - got, 256), 256, 0, h->stream>>>(cand.p, got, np2);
    TN_LAUNCH_CHECK(h);
  }
  for (unsigned k = 2; k <= np2; k <<= 1)
    for (unsigned j = k >> 1; j > 0; j >>= 1) {
      k_lbp_bitonic<<<cdiv(np2, 256), 256, 0, h->stream>>>(cand.p, np2, k, j);
      TN_LAUNCH_CHECK(h);
    }
  const int nk = (int)std::min<i64>(Keff, got);
  std::vector<PS> hc(nk);
  TN_CUDA(cudaMemcpyAsync(hc.data(), cand.p, sizeof(PS) * nk, cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaStreamSynchronize(h->stream));
  for (int i = 0; i < nk; i++) { states[i] = hc[i].st; logp[i] = std::log(hc[i].p); }
  *n_out = nk;
}
