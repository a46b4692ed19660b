// a2-a4(i): boundary-MPS contraction.  PAPER.md:137 (row after row), Sec. III B 1 + Fig. 7
// (sparse diagrams), Sec. III B 2 + Fig. 8 PAPER.md:165-179 (zipper from a left-canonical MPS with the
// trivial connector, truncated SVD keeping chi values, one-site variational passes).
//
// Every chain position j exposes its "dashed box" Theta_j (Fig. 8(c)) as an implicit operator
//     Theta = Lmap^T . Tc . Umap          rows (outer bond, MPO bond), columns (upper physical leg, new bond)
// where Tc is the only large object (state-indexed, built once per position by theta_core / the
// mediating GEMMs) and Lmap / Umap are cheap maps on the skinny side (projector gathers, c_hi fold,
// edge matrices Bh / Bv).  Zipper SVD, variational update and environment update are then all
// "Tc x skinny" / "Tc^T x skinny" DMMA GEMMs.
#include "kernels.cuh"
#include <algorithm>

namespace {

struct PosInfo {
  int kind;   // 0 site, 1 mediating
  int x;
  int wl, wr, pu, pd;
  bool fold;          // site of a lattice without mediating tensors: Bh folded into the left leg
  const CellDev* c;   // site: its cell; med: the left cell
  const CellDev* cr;  // med: the right cell
};

struct ThetaOp {
  const PosInfo* pos = nullptr;
  bool left = false;   // false: built from the right environment; true: from the left one
  int dx = 1, g = 1;   // outer old bond on Theta's rows; new bond inside Theta's columns
  i64 m = 0, n = 0, mk = 0, nk = 0;
  double* Tc = nullptr;
};

struct EvPair { cudaEvent_t a, b; double* dst; };

struct Ctx {
  tn_handle* h;
  int* d_keep = nullptr;      // device: number of singular values kept at the current bond
  int* d_flag = nullptr;      // device: convergence flag
  double* d_stat = nullptr;   // device: [0] running max of (smallest retained sigma / sigma_1)
  double* d_scal = nullptr;   // device scratch scalars
  std::vector<EvPair> evs;
  uint64_t seed = 1;
  void tic(double* dst) {
    EvPair e; e.dst = dst;
    cudaEventCreate(&e.a); cudaEventCreate(&e.b);
    cudaEventRecord(e.a, h->stream);
    evs.push_back(e);
  }
  void toc() { cudaEventRecord(evs.back().b, h->stream); }
  void flush() {
    cudaStreamSynchronize(h->stream);
    for (auto& e : evs) {
      float ms = 0;
      if (cudaEventElapsedTime(&ms, e.a, e.b) == cudaSuccess) *e.dst += ms;
      cudaEventDestroy(e.a); cudaEventDestroy(e.b);
    }
    evs.clear();
  }
  ~Ctx() {   // normally empty (flush() ran); after an exception the pending events are destroyed here
    for (auto& e : evs) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  }
};

std::vector<PosInfo> row_positions(tn_handle* h, int y) {
  std::vector<PosInfo> pos;
  for (int x = 0; x < h->Lx; x++) {
    const CellDev& c = h->cell(y, x);
    PosInfo s;
    s.kind = 0; s.x = x; s.c = &c; s.cr = nullptr;
    s.fold = !h->has_med();
    s.wl = s.fold ? c.bh_rows : c.n_l * c.n_i;
    s.wr = c.n_r * c.n_o;
    s.pu = c.bv_rows;
    s.pd = c.n_d;
    pos.push_back(s);
    if (h->has_med() && x + 1 < h->Lx) {
      const CellDev& cr = h->cell(y, x + 1);
      PosInfo m;
      m.kind = 1; m.x = x; m.c = &c; m.cr = &cr; m.fold = false;
      m.wl = c.n_r * c.n_o;
      m.wr = cr.n_l * cr.n_i;
      m.pu = cr.bd_rows;
      m.pd = c.n_o;
      pos.push_back(m);
    }
  }
  return pos;
}

// ---- skinny GEMMs on Tc ----------------------------------------------------------------------
void tc_apply_N(Ctx& cx, const ThetaOp& op, const double* X, double* Y, int s) {   // Y[mk x s] = Tc X[nk x s]
  cx.tic(&cx.h->st.ms_theta_apply);
  gemm_rm(cx.h, false, false, (int)op.mk, s, (int)op.nk, op.Tc, (int)op.nk, X, s, Y, s);
  cx.toc();
  cx.h->st.flop_theta_apply += 2.0 * op.mk * op.nk * s;
  cx.h->st.bytes_theta_apply += 8.0 * op.mk * op.nk;
  cx.h->st.theta_apply_calls++;
}
void tc_apply_T(Ctx& cx, const ThetaOp& op, const double* Y, double* Z, int s) {   // Z[nk x s] = Tc^T Y[mk x s]
  cx.tic(&cx.h->st.ms_theta_apply);
  gemm_rm(cx.h, true, false, (int)op.nk, s, (int)op.mk, op.Tc, (int)op.nk, Y, s, Z, s);
  cx.toc();
  cx.h->st.flop_theta_apply += 2.0 * op.mk * op.nk * s;
  cx.h->st.bytes_theta_apply += 8.0 * op.mk * op.nk;
  cx.h->st.theta_apply_calls++;
}

// Y[m x s] = Theta X[n x s]
void apply_N(Ctx& cx, const ThetaOp& op, const double* X, double* Y, int s) {
  tn_handle* h = cx.h;
  const PosInfo& p = *op.pos;
  if (p.kind == 1) { tc_apply_N(cx, op, X, Y, s); return; }
  const CellDev& c = *p.c;
  DBuf<double> Xb(h, (size_t)op.nk * s), Yk(h, (size_t)op.mk * s);
  gemm_rm(h, true, false, c.nB, op.g * s, p.pu, c.BvS, c.nB, X, op.g * s, Xb.p, op.g * s);
  tc_apply_N(cx, op, Xb.p, Yk.p, s);
  if (op.left) map_RT(h, c, Yk.p, Y, op.dx, s);
  else map_LT(h, c, p.fold, Yk.p, Y, op.dx, s);
}
// Z[n x s] = Theta^T Y[m x s]
void apply_T(Ctx& cx, const ThetaOp& op, const double* Y, double* Z, int s) {
  tn_handle* h = cx.h;
  const PosInfo& p = *op.pos;
  if (p.kind == 1) { tc_apply_T(cx, op, Y, Z, s); return; }
  const CellDev& c = *p.c;
  DBuf<double> Yk(h, (size_t)op.mk * s), Zb(h, (size_t)op.nk * s);
  if (op.left) map_R(h, c, Y, Yk.p, op.dx, s);
  else map_L(h, c, p.fold, Y, Yk.p, op.dx, s);
  tc_apply_T(cx, op, Yk.p, Zb.p, s);
  gemm_rm(h, false, false, p.pu, op.g * s, c.nB, c.BvS, c.nB, Zb.p, op.g * s, Z, op.g * s);
}

// ---- Theta build -----------------------------------------------------------------------------
// A: old MPS tensor [al][pd][ar]; E: environment on the far side, [(dy, w), g]
ThetaOp build_op(Ctx& cx, const PosInfo& p, bool left, const MpsTensor& A, const double* E, int g) {
  tn_handle* h = cx.h;
  ThetaOp op;
  op.pos = &p; op.left = left; op.g = g;
  const int al = A.dl, ar = A.dr;
  op.dx = left ? ar : al;
  const int dy = left ? al : ar;
  cx.tic(&h->st.ms_theta_build);
  if (p.kind == 0) {
    const CellDev& c = *p.c;
    op.m = (i64)op.dx * (left ? p.wr : p.wl);
    op.n = (i64)p.pu * g;
    op.mk = (i64)op.dx * c.nK;
    op.nk = (i64)c.nB * g;
    op.Tc = h->dalloc<double>((size_t)op.mk * op.nk);
    DBuf<double> Ek(h, (size_t)dy * c.nK * g);
    if (left) {
      map_L(h, c, p.fold, E, Ek.p, dy, g);
      DBuf<double> At(h, (size_t)al * A.p * ar);
      permute3(h, At.p, A.d, ar, A.p, al, 1, ar, (i64)A.p * ar);
      theta_core(h, c, At.p, op.dx, dy, Ek.p, g, op.Tc);
    } else {
      map_R(h, c, E, Ek.p, dy, g);
      theta_core(h, c, A.d, op.dx, dy, Ek.p, g, op.Tc);
    }
  } else {
    const CellDev& cl = *p.c;
    const CellDev& cr = *p.cr;
    const int n_r = cl.n_r, n_o = cl.n_o, n_lp = cr.n_l, n_i = cr.n_i, n_q = cr.bd_rows;
    if (!left) {
      op.m = op.mk = (i64)al * n_r * n_o;
      op.n = op.nk = (i64)n_q * g;
      op.Tc = h->dalloc<double>((size_t)op.mk * op.nk);
      DBuf<double> Rm2(h, (size_t)ar * n_r * n_i * g), T1(h, (size_t)al * n_o * n_r * n_i * g);
      GemmDesc d;
      d.B1 = ar; d.M = n_r; d.N = n_i * g; d.K = n_lp;
      d.A = cr.Bh; d.a_i = n_lp; d.a_k = 1;
      d.B = E; d.b_b1 = (i64)n_lp * n_i * g; d.b_k = (i64)n_i * g; d.b_j = 1;
      d.C = Rm2.p; d.c_b1 = (i64)n_r * n_i * g; d.c_i = (i64)n_i * g; d.c_j = 1;
      d.nsplit = 1;
      gemm_general(h, d);
      gemm_rm(h, false, false, al * n_o, n_r * n_i * g, ar, A.d, ar, Rm2.p, n_r * n_i * g, T1.p, n_r * n_i * g);
      med_apply_bd(h, T1.p, cr.Bd, op.Tc, al, n_o, n_r, n_i, n_q, g);
      h->st.flop_theta_build += 2.0 * ar * n_r * n_i * g * n_lp + 2.0 * al * n_o * (double)n_r * n_i * g * ar +
                                2.0 * (double)op.mk * op.nk * n_i;
    } else {
      op.m = op.mk = (i64)ar * n_lp * n_i;
      op.n = op.nk = (i64)n_q * g;
      op.Tc = h->dalloc<double>((size_t)op.mk * op.nk);
      DBuf<double> Lk(h, (size_t)n_lp * al * n_o * g), TL(h, (size_t)ar * n_lp * g);
      GemmDesc d;
      d.B1 = al; d.B2 = n_o; d.M = n_lp; d.N = g; d.K = n_r;
      d.A = cr.Bh; d.a_i = 1; d.a_k = n_lp;
      d.B = E; d.b_b1 = (i64)n_r * n_o * g; d.b_b2 = g; d.b_k = (i64)n_o * g; d.b_j = 1;
      d.C = Lk.p; d.c_b1 = (i64)n_o * g; d.c_b2 = g; d.c_i = (i64)al * n_o * g; d.c_j = 1;
      d.nsplit = 1;
      gemm_general(h, d);
      GemmDesc e;
      e.B1 = n_lp; e.M = ar; e.N = g; e.K = al * n_o;
      e.A = A.d; e.a_i = 1; e.a_k = ar;
      e.B = Lk.p; e.b_b1 = (i64)al * n_o * g; e.b_k = g; e.b_j = 1;
      e.C = TL.p; e.c_b1 = g; e.c_i = (i64)n_lp * g; e.c_j = 1;
      e.nsplit = 1;
      gemm_general(h, e);
      med_outer_bd(h, TL.p, cr.Bd, op.Tc, (i64)ar * n_lp, n_i, n_q, g);
      h->st.flop_theta_build += 2.0 * al * n_o * (double)n_lp * g * n_r + 2.0 * n_lp * (double)ar * g * al * n_o;
    }
  }
  cx.toc();
  return op;
}
void free_op(Ctx& cx, ThetaOp& op) {
  if (op.Tc) cx.h->dfree(op.Tc);
  op.Tc = nullptr;
}

// ---- truncated SVD of the implicit Theta: block subspace iteration + Rayleigh-Ritz -----------
__global__ void k_rank_decide(const double* sig, int ks, int chi, int gap_guard, int* keep, double* stat) {
  if (threadIdx.x || blockIdx.x) return;
  double s0 = sig[0];
  int k = 0;
  if (s0 > 0.0)
    for (int i = 0; i < ks; i++) k += sig[i] > 1e-14 * s0 ? 1 : 0;
  bool cut = false;
  if (k > chi) {
    cut = true;
    k = chi;
    if (gap_guard)
      while (k > 1 && sig[k] >= (1.0 - 1e-6) * sig[k - 1]) k--;
  }
  if (k < 1) k = 1;
  *keep = k;
  stat[1] = (cut && s0 > 0.0) ? sig[k - 1] / s0 : 0.0;   // only bonds that really truncate; committed at convergence
}
__global__ void k_commit_stat(double* stat) {
  if (threadIdx.x || blockIdx.x) return;
  stat[0] = fmax(stat[0], stat[1]);
}
// Range bookkeeping (reading S19): *safe = (*s > 0 ? *s : 1), *ls_out = (ls_in ? *ls_in : 0) + log(*safe)
__global__ void k_ls_step(const double* s, const double* ls_in, double* ls_out, double* safe) {
  if (threadIdx.x || blockIdx.x) return;
  double v = *s;
  if (!(v > 0.0) || !isfinite(v)) v = 1.0;
  *safe = v;
  *ls_out = (ls_in ? *ls_in : 0.0) + log(v);
}
// partial column sums of squares of (P - Q), both [m x k]: block (32 columns x 8 row lanes), fixed reduction order
__global__ void __launch_bounds__(256) k_coldiff_part(const double* P, const double* Q, i64 m, int k, int rows_per_block,
                                                      double* part) {
  __shared__ double sh[8][33];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const i64 r0 = (i64)blockIdx.x * rows_per_block, r1 = min(m, r0 + rows_per_block);
  for (int c0 = 0; c0 < k; c0 += 32) {
    const int col = c0 + tx;
    double s = 0.0;
    if (col < k)
      for (i64 r = r0 + ty; r < r1; r += 8) {
        double d = P[r * k + col] - Q[r * k + col];
        s += d * d;
      }
    sh[ty][tx] = s;
    __syncthreads();
    if (ty == 0 && col < k) {
      double t = 0.0;
#pragma unroll
      for (int y = 0; y < 8; y++) t += sh[y][tx];
      part[(i64)blockIdx.x * k + col] = t;
    }
    __syncthreads();
  }
}
struct SvdInfo { int flag, keep; double res, sig0, sigk, sigl; };   // device -> host once per iteration
// flag = every kept triplet has residual <= tol sigma_1; res = worst residual / (tol sigma_1);
// sig0 / sigk / sigl = largest, smallest kept and smallest Ritz value of the block (they steer the Chebyshev filter)
__global__ void k_resid_flag(const double* part, int nblk, int k, const int* keep, const double* sig, double tol,
                             int* flag, SvdInfo* info, double* res_out, int col0) {
  __shared__ int bad;
  __shared__ double worst[1024];   // one slot per thread: the block has up to 1024 threads (exact mode: k up to TN_OPT_EXACT_CAP)
  if (threadIdx.x == 0) bad = 0;
  __syncthreads();
  // columns of this block are columns col0 .. col0 + k - 1 of the full Ritz list; sig points at the FULL list
  int col = threadIdx.x;
  double w = 0.0;
  if (col < k) {
    double s = 0.0;
    for (int b = 0; b < nblk; b++) s += part[(i64)b * k + col];
    w = sig[0] > 0.0 ? sqrt(s) / (tol * sig[0]) : 0.0;
    if (!(w == w)) w = 1e300;
    if (res_out) res_out[col] = w;
    if (col0 + col < *keep) { if (!(w <= 1.0)) bad = 1; } else w = 0.0;
  }
  worst[threadIdx.x] = w;
  __syncthreads();
  if (threadIdx.x == 0) {
    double mx = 0.0;
    for (int i = 0; i < (int)blockDim.x; i++) mx = fmax(mx, worst[i]);
    *flag = bad ? 0 : 1;
    info->flag = bad ? 0 : 1; info->keep = *keep; info->res = mx;
    info->sig0 = sig[0]; info->sigk = sig[max(0, *keep - 1)]; info->sigl = sig[col0 + k - 1];
  }
}
// Chebyshev recurrence step on the block:  Fn = alpha (W - cm F) + beta Fp
__global__ void k_cheb_step(double* Fn, const double* W, const double* F, const double* Fp, i64 n, double alpha, double cm,
                            double beta) {
  i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) Fn[i] = alpha * (W[i] - cm * F[i]) + (Fp ? beta * Fp[i] : 0.0);
}

// ---- helpers of the locked iteration -----------------------------------------------------------------------
// dst[r][dc0 + j] = src[r][sc0 + j] * (inv_scale ? 1 / inv_scale[j] : 1),  j < nc
__global__ void k_copy_cols(double* dst, int ldd, int dc0, const double* src, int lds, int sc0, i64 rows, int nc,
                            const double* inv_scale) {
  i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= rows * nc) return;
  const i64 r = t / nc;
  const int j = (int)(t % nc);
  double v = src[r * lds + sc0 + j];
  if (inv_scale) { const double s = inv_scale[j]; v = s > 0.0 ? v / s : 0.0; }
  dst[r * ldd + dc0 + j] = v;
}
__global__ void k_sub(double* Y, const double* P, i64 n) {
  i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) Y[i] -= P[i];
}
static void copy_cols(tn_handle* h, double* dst, int ldd, int dc0, const double* src, int lds, int sc0, i64 rows, int nc,
                      const double* inv_scale = nullptr) {
  if (rows <= 0 || nc <= 0) return;
  k_copy_cols<<<cdiv(rows * nc, 256), 256, 0, h->stream>>>(dst, ldd, dc0, src, lds, sc0, rows, nc, inv_scale);
  TN_LAUNCH_CHECK(h);
}
// X[rows x s] -= Q[:, :L] (Q[:, :L]^T X)   (Q has leading dimension ldq; one classical Gram-Schmidt pass)
static void project_out(tn_handle* h, double* X, i64 rows, int s, const double* Q, int ldq, int L, double* coef, double* tmp) {
  if (L <= 0) return;
  gemm_rm(h, true, false, L, s, (int)rows, Q, ldq, X, s, coef, s);
  gemm_rm(h, false, false, (int)rows, s, L, Q, ldq, coef, s, tmp, s);
  k_sub<<<cdiv(rows * s, 256), 256, 0, h->stream>>>(X, tmp, rows * s);
  TN_LAUNCH_CHECK(h);
}

// Truncated SVD of the implicit Theta by block subspace iteration WITH LOCKING (deflation): the leading Ritz
// triplets converge first (rate (sigma_{ks+1} / sigma_i)^2 per iteration), so once an even-sized prefix of the
// active block has residual <= tol sigma_1 it is frozen (V_lock, U_lock = Theta V_lock / sigma) and the following
// iterations apply Theta only to the remaining columns, kept orthogonal to the frozen ones by one projection per
// apply.  Same converged subspace and the same test as the plain iteration (reading S1); measured on a D = 64,
// h = 0 Pegasus-shaped slice the plain iteration spends 53 % of its column-applies on already converged columns.
// (A Chebyshev filter on the deflated active block was measured too: it locks later and costs 10-16 % MORE
// FLOP than locking alone, so the filter stays with the non-locked fallback below.)
void svd_trunc_locked(Ctx& cx, const ThetaOp& op, int chi, int ks, double* Vz, double* C, double* sig0_out) {
  tn_handle* h = cx.h;
  const i64 m = op.m, n = op.n;
  const int ldl = ks;
  DBuf<double> Om(h, (size_t)n * ks), Z(h, (size_t)n * ks), Vrot(h, (size_t)n * ks), Vl(h, (size_t)n * ldl);
  DBuf<double> Ya(h, (size_t)m * ks), Yb(h, (size_t)m * ks), TV(h, (size_t)m * ks), US(h, (size_t)m * ks);
  DBuf<double> Ul(h, (size_t)m * ldl), CL(h, (size_t)m * ldl);
  DBuf<double> B(h, (size_t)ks * ks), Bo(h, (size_t)ks * ks), Wt(h, (size_t)ks * ks), coef(h, (size_t)ks * ks);
  DBuf<double> sigfull(h, ks), dres(h, 128);
  DBuf<SvdInfo> dinfo(h, 1);
  double* Y = Ya.p;
  double* Yn = Yb.p;
  fill_random(h, Om.p, n * ks, cx.seed++);
  cx.tic(&h->st.ms_orth_svd);
  orth_columns(h, Om.p, n, ks, 3);
  cx.toc();
  const int rpb = (int)std::max<i64>(64, (m + 255) / 256);
  const int nblk = cdiv(m, rpb);
  DBuf<double> part(h, (size_t)nblk * ks);
  std::vector<double> res(128, 0.0);
  int L = 0, sa = ks;
  bool have_rr = false;
  // skip the first Rayleigh-Ritz step / test when the previous SVD of this contraction did not converge at its
  // first test (a random start block needs >= 2 power steps unless Theta is rank-deficient below ks, config 5)
  const bool skip_first_rr = h->svd_skip_first && ks < std::min(m, n);
  int n_rr = 0;
  double last_res = 1.0;
  for (int it = 0;; it++) {
    apply_N(cx, op, Om.p, Yn, sa);
    if (have_rr) {
      gemm_rm(h, false, true, (int)m, sa, sa, Yn, sa, Wt.p, sa, TV.p, sa);      // Theta V_a
      gemm_rm(h, false, true, (int)m, sa, sa, Y, sa, Bo.p, sa, US.p, sa);       // U_a Sigma_a
      k_coldiff_part<<<nblk, 256, 0, h->stream>>>(TV.p, US.p, m, sa, rpb, part.p);
      TN_LAUNCH_CHECK(h);
      k_resid_flag<<<1, std::max(32, (sa + 31) / 32 * 32), 0, h->stream>>>(part.p, nblk, sa, cx.d_keep, sigfull.p,
                                                                        h->svd_tol, cx.d_flag, dinfo.p, dres.p, L);
      TN_LAUNCH_CHECK(h);
      SvdInfo info;
      TN_CUDA(cudaMemcpyAsync(&info, dinfo.p, sizeof(info), cudaMemcpyDeviceToHost, h->stream));
      TN_CUDA(cudaMemcpyAsync(res.data(), dres.p, sizeof(double) * sa, cudaMemcpyDeviceToHost, h->stream));
      TN_CUDA(cudaStreamSynchronize(h->stream));
      last_res = info.res;
      if (info.flag) break;
      if (it >= h->svd_maxit) { h->st.svd_unconverged++; break; }
      int c = 0;
      while (c < sa && res[c] <= 1.0) c++;
      c = std::min(c, std::max(0, info.keep - L)) & ~1;
      if (c >= 4 && sa - c >= 8) {   // freeze the converged prefix
        gemm_rm(h, false, true, (int)n, sa, sa, Om.p, sa, Wt.p, sa, Vrot.p, sa);   // V_a = Om W
        copy_cols(h, Vl.p, ldl, L, Vrot.p, sa, 0, n, c);
        copy_cols(h, CL.p, ldl, L, TV.p, sa, 0, m, c);
        copy_cols(h, Ul.p, ldl, L, TV.p, sa, 0, m, c, sigfull.p + L);
        copy_cols(h, Om.p, sa - c, 0, Vrot.p, sa, c, n, sa - c);
        copy_cols(h, Yn, sa - c, 0, TV.p, sa, c, m, sa - c);                       // Theta V_a of the rest: already known
        L += c;
        sa -= c;
        h->st.svd_locked_cols += c;
      }
    }
    std::swap(Y, Yn);
    project_out(h, Y, m, sa, Ul.p, ldl, L, coef.p, US.p);
    cx.tic(&h->st.ms_orth_svd);
    orth_columns(h, Y, m, sa, 5);
    cx.toc();
    apply_T(cx, op, Y, Z.p, sa);
    project_out(h, Z.p, n, sa, Vl.p, ldl, L, coef.p, Vrot.p);
    TN_CUDA(cudaMemcpyAsync(Om.p, Z.p, sizeof(double) * n * sa, cudaMemcpyDeviceToDevice, h->stream));
    cx.tic(&h->st.ms_orth_svd);
    orth_columns(h, Om.p, n, sa, 5);
    h->st.svd_iterations++;
    if (it == 0 && skip_first_rr) {   // a random start block is never converged after one step: no Rayleigh-Ritz, no test
      cx.toc();
      continue;
    }
    gemm_rm(h, true, false, sa, sa, (int)n, Om.p, sa, Z.p, sa, B.p, sa);
    jacobi_rows(h, B.p, sa, sa, sa, Bo.p, Wt.p, sigfull.p + L);
    k_rank_decide<<<1, 32, 0, h->stream>>>(sigfull.p, L + sa, chi, h->gap_guard, cx.d_keep, cx.d_stat);
    TN_LAUNCH_CHECK(h);
    cx.toc();
    have_rr = true;
    n_rr++;
  }
  if (!skip_first_rr) h->svd_skip_first = n_rr >= 2;
  else if (n_rr == 1 && last_res < 1e-3) h->svd_skip_first = 0;
  k_commit_stat<<<1, 32, 0, h->stream>>>(cx.d_stat);
  TN_LAUNCH_CHECK(h);
  gemm_rm(h, false, true, (int)n, sa, sa, Om.p, sa, Wt.p, sa, Vrot.p, sa);          // V_a = Om W
  const int kt = L + sa;
  copy_cols(h, Z.p, kt, 0, Vl.p, ldl, 0, n, L);
  copy_cols(h, Z.p, kt, L, Vrot.p, sa, 0, n, sa);
  copy_cols(h, US.p, kt, 0, CL.p, ldl, 0, m, L);
  copy_cols(h, US.p, kt, L, TV.p, sa, 0, m, sa);
  permute3(h, Vz, Z.p, 1, (int)n, chi, 0, kt, 1, 2, cx.d_keep);
  permute3(h, C, US.p, 1, (int)m, chi, 0, kt, 1, 2, cx.d_keep);
  TN_CUDA(cudaMemcpyAsync(sig0_out, sigfull.p, sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
}

// Outputs: Vz [n x chi] leading right singular vectors, C [m x chi] = Theta Vz; columns >= keep are zero.
void svd_trunc(Ctx& cx, const ThetaOp& op, int chi, int ks, double* Vz, double* C, double* sig0_out) {
  tn_handle* h = cx.h;
  const i64 m = op.m, n = op.n;
  if (h->svd_lock && ks <= 96 && (ks & 1) == 0 && chi < ks && ks >= 24) {
    svd_trunc_locked(cx, op, chi, ks, Vz, C, sig0_out);
    return;
  }
  if (ks > 1024) tn_throw(TN_ERR_ARG, "truncated SVD block of %d columns: at most 1024 are supported", ks);
  DBuf<double> Om(h, (size_t)n * ks), Z(h, (size_t)n * ks), Ya(h, (size_t)m * ks), Yb(h, (size_t)m * ks);
  DBuf<double> TV(h, (size_t)m * ks), US(h, (size_t)m * ks);
  DBuf<double> B(h, (size_t)ks * ks), Bo(h, (size_t)ks * ks), Wt(h, (size_t)ks * ks), sig(h, ks);
  double* Y = Ya.p;
  double* Yn = Yb.p;
  fill_random(h, Om.p, n * ks, cx.seed++);
  cx.tic(&h->st.ms_orth_svd);
  orth_columns(h, Om.p, n, ks, 3);
  cx.toc();
  const int rpb = (int)std::max<i64>(64, (m + 255) / 256);
  const int nblk = cdiv(m, rpb);
  DBuf<double> part(h, (size_t)nblk * ks);
  DBuf<SvdInfo> dinfo(h, 1);
  bool prev = false;
  const bool skip_first_rr = h->svd_skip_first && ks < std::min(m, n);
  int n_rr = 0;
  double last_res = 1.0;
  for (int it = 0;; it++) {
    apply_N(cx, op, Om.p, Yn, ks);
    if (prev) {
      gemm_rm(h, false, true, (int)m, ks, ks, Yn, ks, Wt.p, ks, TV.p, ks);
      gemm_rm(h, false, true, (int)m, ks, ks, Y, ks, Bo.p, ks, US.p, ks);
      k_coldiff_part<<<nblk, 256, 0, h->stream>>>(TV.p, US.p, m, ks, rpb, part.p);
      TN_LAUNCH_CHECK(h);
      k_resid_flag<<<1, std::max(32, (ks + 31) / 32 * 32), 0, h->stream>>>(part.p, nblk, ks, cx.d_keep, sig.p,
                                                                        h->svd_tol, cx.d_flag, dinfo.p, nullptr, 0);
      TN_LAUNCH_CHECK(h);
      SvdInfo info;
      TN_CUDA(cudaMemcpyAsync(&info, dinfo.p, sizeof(info), cudaMemcpyDeviceToHost, h->stream));
      TN_CUDA(cudaStreamSynchronize(h->stream));
      last_res = info.res;
      if (info.flag) break;
      if (it >= h->svd_maxit) { h->st.svd_unconverged++; break; }
      // ---- Chebyshev-filtered step: when the worst residual is still far from the tolerance
      // and the block's Ritz values decay slowly, replace the plain power step by T_d((A - b/2) / (b/2)) Om with
      // A = Theta^T Theta and [0, b] = the unwanted part of the spectrum (b = smallest Ritz value^2 of the block).
      // Same subspace, same convergence test, fewer applies; d is capped so that the amplification of sigma_1
      // stays below 1e20 (fast-decaying spectra fall back to d = 1 = the plain step).
      const double lam1 = info.sig0 * info.sig0, lamk = info.sigk * info.sigk, b = info.sigl * info.sigl;
      int deg = 1;
      const double cheb_cap = 1e20;   // measured on a D = 64, h = 0 Pegasus-shaped slice: 1e13 never engages, 1e30 loses the small directions
      const double res_min = 1e2, gap_max = 30.0;
      const int deg_max = 6;
      if (h->svd_cheb && info.res > res_min && b > 1e-20 * lam1 && lamk < gap_max * b) {
        const double x1 = 2.0 * lam1 / b - 1.0;
        deg = (int)std::floor(std::log(2.0 * cheb_cap) / std::log(x1 + std::sqrt(x1 * x1 - 1.0)));
        deg = std::min(deg, deg_max);
      }
      if (deg >= 2) {
        const double cm = 0.5 * b, e = 0.5 * b;
        const i64 ne = n * ks;
        DBuf<double> F1(h, (size_t)ne), F2(h, (size_t)ne);
        double* ring[3] = {Om.p, F1.p, F2.p};   // F_0 = Om lives in ring[0]
        int ip = -1, ic = 0, in = 1;
        apply_T(cx, op, Yn, Z.p, ks);           // A F_0 = Theta^T (Theta Om): Yn is already in hand
        for (int j = 0; j < deg; j++) {
          if (j > 0) {
            apply_N(cx, op, ring[ic], Yn, ks);
            apply_T(cx, op, Yn, Z.p, ks);
          }
          k_cheb_step<<<cdiv(ne, 256), 256, 0, h->stream>>>(ring[in], Z.p, ring[ic], ip >= 0 ? ring[ip] : nullptr, ne,
                                                           (j == 0 ? 1.0 : 2.0) / e, cm, -1.0);
          TN_LAUNCH_CHECK(h);
          const int free_ = ip >= 0 ? ip : 2;
          ip = ic; ic = in; in = free_;
        }
        double* Fc = ring[ic];
        if (Fc != Om.p) TN_CUDA(cudaMemcpyAsync(Om.p, Fc, sizeof(double) * ne, cudaMemcpyDeviceToDevice, h->stream));
        cx.tic(&h->st.ms_orth_svd);
        orth_columns(h, Om.p, n, ks, 5);
        cx.toc();
        prev = false;
        h->st.cheb_steps += deg;
        continue;
      }
    }
    std::swap(Y, Yn);
    cx.tic(&h->st.ms_orth_svd);
    orth_columns(h, Y, m, ks, 5);
    cx.toc();
    apply_T(cx, op, Y, Z.p, ks);
    TN_CUDA(cudaMemcpyAsync(Om.p, Z.p, sizeof(double) * n * ks, cudaMemcpyDeviceToDevice, h->stream));
    cx.tic(&h->st.ms_orth_svd);
    orth_columns(h, Om.p, n, ks, 5);
    h->st.svd_iterations++;
    if (it == 0 && skip_first_rr) {   // random start block: skip the first Rayleigh-Ritz step and its test
      cx.toc();
      continue;
    }
    gemm_rm(h, true, false, ks, ks, (int)n, Om.p, ks, Z.p, ks, B.p, ks);
    jacobi_rows(h, B.p, ks, ks, ks, Bo.p, Wt.p, sig.p);
    k_rank_decide<<<1, 32, 0, h->stream>>>(sig.p, ks, chi, h->gap_guard, cx.d_keep, cx.d_stat);
    TN_LAUNCH_CHECK(h);
    cx.toc();
    prev = true;
    n_rr++;
  }
  if (!skip_first_rr) h->svd_skip_first = n_rr >= 2;
  else if (n_rr == 1 && last_res < 1e-3) h->svd_skip_first = 0;
  k_commit_stat<<<1, 32, 0, h->stream>>>(cx.d_stat);
  TN_LAUNCH_CHECK(h);
  gemm_rm(h, false, true, (int)n, ks, ks, Om.p, ks, Wt.p, ks, Z.p, ks);        // V = Omega W
  permute3(h, Vz, Z.p, 1, (int)n, chi, 0, ks, 1, 2, cx.d_keep);
  permute3(h, C, TV.p, 1, (int)m, chi, 0, ks, 1, 2, cx.d_keep);
  TN_CUDA(cudaMemcpyAsync(sig0_out, sig.p, sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
}

// Truncated randomized SVD (TN_OPT_SVD_MODE = 1, refs [43, 44]): `iters` subspace iterations from a
// seeded, counter-based random block, one Rayleigh-Ritz step, no convergence test (so no host round trip):
//   Om <- orth(Omega);  iters x { Y <- orth(Theta Om);  Z <- Theta^T Y;  Om <- orth(Z) };  B = Om^T Z = W S X^T;  V = Om W.
// Outputs as svd_trunc: Vz [n x chi] leading Ritz vectors, C [m x chi] = Theta Vz; columns >= keep are zero.
void svd_rand(Ctx& cx, const ThetaOp& op, int chi, int ks, int pu, int g, double* Vz, double* C, double* sig0_out) {
  tn_handle* h = cx.h;
  const i64 m = op.m, n = op.n;
  if (ks > 1024 || g > 4096) tn_throw(TN_ERR_ARG, "randomized SVD block of %d columns / bond %d: at most 1024 / 4096", ks, g);
  DBuf<double> Om(h, (size_t)n * ks), Z(h, (size_t)n * ks), Y(h, (size_t)m * ks);
  DBuf<double> B(h, (size_t)ks * ks), Bo(h, (size_t)ks * ks), Wt(h, (size_t)ks * ks), sig(h, ks);
  fill_random_pgc(h, Om.p, pu, g, ks, cx.seed++);
  cx.tic(&h->st.ms_orth_svd);
  orth_columns(h, Om.p, n, ks, 3);
  cx.toc();
  for (int it = 0; it < std::max(1, h->rsvd_iters); it++) {
    apply_N(cx, op, Om.p, Y.p, ks);
    cx.tic(&h->st.ms_orth_svd);
    orth_columns(h, Y.p, m, ks, 5);
    cx.toc();
    apply_T(cx, op, Y.p, Z.p, ks);
    TN_CUDA(cudaMemcpyAsync(Om.p, Z.p, sizeof(double) * n * ks, cudaMemcpyDeviceToDevice, h->stream));
    cx.tic(&h->st.ms_orth_svd);
    orth_columns(h, Om.p, n, ks, 5);
    cx.toc();
    h->st.svd_iterations++;
  }
  cx.tic(&h->st.ms_orth_svd);
  gemm_rm(h, true, false, ks, ks, (int)n, Om.p, ks, Z.p, ks, B.p, ks);
  jacobi_rows(h, B.p, ks, ks, ks, Bo.p, Wt.p, sig.p);
  k_rank_decide<<<1, 32, 0, h->stream>>>(sig.p, ks, chi, h->gap_guard, cx.d_keep, cx.d_stat);
  TN_LAUNCH_CHECK(h);
  k_commit_stat<<<1, 32, 0, h->stream>>>(cx.d_stat);
  TN_LAUNCH_CHECK(h);
  cx.toc();
  gemm_rm(h, false, true, (int)n, ks, ks, Om.p, ks, Wt.p, ks, Z.p, ks);        // V = Om W
  permute3(h, Vz, Z.p, 1, (int)n, chi, 0, ks, 1, 2, cx.d_keep);
  apply_N(cx, op, Vz, C, chi);                                                  // connector = Theta V (exact for this V)
  TN_CUDA(cudaMemcpyAsync(sig0_out, sig.p, sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
}

// Tiny Theta (both dimensions of the order of 100: every position of the one-spin-per-site square lattice, the first
// and last positions of any row, config 1): the matrix is formed explicitly by one apply to the identity and decomposed
// by the one-sided Jacobi kernel -- an exact SVD in ~6 launches, no iteration and no host round trip, where the subspace
// iteration needs ~40 launches and a device -> host flag per step.  Same outputs as svd_trunc.
__global__ void k_eye(double* X, int n) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n * n) X[t] = (t / n == t % n) ? 1.0 : 0.0;
}
bool svd_direct_fits(i64 m, i64 n) { return n <= 128 && m <= 4096 && n * m + n * n <= 24000; }
void svd_direct(Ctx& cx, const ThetaOp& op, int chi, double* Vz, double* C, double* sig0_out) {
  tn_handle* h = cx.h;
  const int m = (int)op.m, n = (int)op.n;
  DBuf<double> X(h, (size_t)n * n), Th(h, (size_t)m * n), ThT(h, (size_t)n * m), Mo(h, (size_t)n * m), Wt(h, (size_t)n * n), sig(h, n);
  cx.seed++;                                                     // one seed per truncated SVD, whichever route takes it
  k_eye<<<cdiv((i64)n * n, 256), 256, 0, h->stream>>>(X.p, n);
  TN_LAUNCH_CHECK(h);
  apply_N(cx, op, X.p, Th.p, n);                                 // Theta [m x n]
  cx.tic(&h->st.ms_orth_svd);
  permute3(h, ThT.p, Th.p, 1, n, m, 0, 1, n);                    // Theta^T [n x m]
  jacobi_rows(h, ThT.p, m, n, m, Mo.p, Wt.p, sig.p);             // rows of V^T Theta^T orthogonal: Wt = V^T, Mo = (Theta V)^T
  k_rank_decide<<<1, 32, 0, h->stream>>>(sig.p, std::min(m, n), chi, h->gap_guard, cx.d_keep, cx.d_stat);
  TN_LAUNCH_CHECK(h);
  k_commit_stat<<<1, 32, 0, h->stream>>>(cx.d_stat);
  TN_LAUNCH_CHECK(h);
  cx.toc();
  permute3(h, Vz, Wt.p, 1, n, chi, 0, 1, n, 2, cx.d_keep);
  permute3(h, C, Mo.p, 1, m, chi, 0, 1, m, 2, cx.d_keep);
  TN_CUDA(cudaMemcpyAsync(sig0_out, sig.p, sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
  h->st.svd_direct++;
}

MpsTensor new_tensor(tn_handle* h, int dl, int p, int dr) {
  MpsTensor t;
  t.dl = dl; t.p = p; t.dr = dr;
  t.d = h->dalloc<double>((size_t)dl * p * dr);
  return t;
}

// C-1: QR chain left -> right on T in place (Fig. 8(c) "initial MPS in the left canonical form"); *rlast = the final 1 x 1 factor
void left_canonicalize(Ctx& cx, std::vector<MpsTensor>& A, double* rlast) {
  tn_handle* h = cx.h;
  const int n = (int)A.size();
  for (int j = 0; j < n; j++) {
    const i64 rows = (i64)A[j].dl * A[j].p;
    const int ar = A[j].dr;
    DBuf<double> Q(h, (size_t)rows * ar), Rf(h, (size_t)ar * ar);
    TN_CUDA(cudaMemcpyAsync(Q.p, A[j].d, sizeof(double) * rows * ar, cudaMemcpyDeviceToDevice, h->stream));
    cx.tic(&h->st.ms_orth_svd);
    orth_columns(h, Q.p, rows, ar, 5);
    cx.toc();
    gemm_rm(h, true, false, ar, ar, (int)rows, Q.p, ar, A[j].d, ar, Rf.p, ar);
    TN_CUDA(cudaMemcpyAsync(A[j].d, Q.p, sizeof(double) * rows * ar, cudaMemcpyDeviceToDevice, h->stream));
    if (j + 1 < n) {
      const int cols = A[j + 1].p * A[j + 1].dr;
      DBuf<double> T(h, (size_t)ar * cols);
      gemm_rm(h, false, false, ar, cols, ar, Rf.p, ar, A[j + 1].d, cols, T.p, cols);
      TN_CUDA(cudaMemcpyAsync(A[j + 1].d, T.p, sizeof(double) * ar * cols, cudaMemcpyDeviceToDevice, h->stream));
    } else {
      TN_CUDA(cudaMemcpyAsync(rlast, Rf.p, sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    }
  }
}

// Second step of the two-step truncation 2 chi -> chi: canonical compression of the unit-norm MPS N to
// bond <= D (left-canonicalise, then LQ + small SVD at every bond right -> left; rank / gap rules as in the zipper).
// N is replaced; *nu (device) receives the norm left after the cut.
void truncate_mps(Ctx& cx, std::vector<MpsTensor>& N, int D, double* nu) {
  tn_handle* h = cx.h;
  const int n = (int)N.size();
  DBuf<double> rl(h, 1);
  left_canonicalize(cx, N, rl.p);
  scale_by(h, N[n - 1].d, (i64)N[n - 1].dl * N[n - 1].p * N[n - 1].dr, rl.p, false);
  for (int j = n - 1; j >= 1; j--) {
    const int dl = N[j].dl, pc = N[j].p * N[j].dr;            // M = N[j] as [dl x pc]
    const int kn = std::min(D, std::min(dl, pc));             // static new bond
    DBuf<double> Qt(h, (size_t)pc * dl), L(h, (size_t)dl * dl), Lt(h, (size_t)dl * dl), Mo(h, (size_t)dl * dl);
    DBuf<double> Wt(h, (size_t)dl * dl), sig(h, dl), T(h, (size_t)pc * dl);
    permute3(h, Qt.p, N[j].d, 1, pc, dl, 0, 1, pc);           // Qt = M^T [pc x dl]
    cx.tic(&h->st.ms_orth_svd);
    orth_columns(h, Qt.p, pc, dl, 5);                         // M = L Qt^T with Qt^T right-canonical
    gemm_rm(h, false, false, dl, dl, pc, N[j].d, pc, Qt.p, dl, L.p, dl);
    permute3(h, Lt.p, L.p, 1, dl, dl, 0, 1, dl);
    jacobi_rows(h, Lt.p, dl, dl, dl, Mo.p, Wt.p, sig.p);      // L = U S X^T:  Mo = S U^T,  Wt = X^T
    k_rank_decide<<<1, 32, 0, h->stream>>>(sig.p, dl, kn, h->gap_guard, cx.d_keep, cx.d_stat);
    TN_LAUNCH_CHECK(h);
    k_commit_stat<<<1, 32, 0, h->stream>>>(cx.d_stat);
    TN_LAUNCH_CHECK(h);
    cx.toc();
    gemm_rm(h, false, true, pc, dl, dl, Qt.p, dl, Wt.p, dl, T.p, dl);          // T = Qt X  [pc x dl]
    MpsTensor nj = new_tensor(h, kn, N[j].p, N[j].dr);
    permute3(h, nj.d, T.p, kn, pc, 1, 1, dl, 0, 0, cx.d_keep);                 // N'[j] = (first kn columns of T)^T, rows >= keep zero
    // carry U S into the left neighbour: N[j-1] [rows x dl] . (Mo^T)[:, :kn]
    const i64 rows = (i64)N[j - 1].dl * N[j - 1].p;
    MpsTensor nl = new_tensor(h, N[j - 1].dl, N[j - 1].p, kn);
    DBuf<double> Tl(h, (size_t)rows * kn);
    gemm_rm(h, false, true, (int)rows, kn, dl, N[j - 1].d, dl, Mo.p, dl, Tl.p, kn);
    permute3(h, nl.d, Tl.p, 1, (int)rows, kn, 0, kn, 1, 2, cx.d_keep);
    h->dfree(N[j].d); h->dfree(N[j - 1].d);
    N[j] = nj; N[j - 1] = nl;
  }
  const i64 n0 = (i64)N[0].dl * N[0].p * N[0].dr;
  frob_norm(h, N[0].d, n0, nu);
  scale_by(h, N[0].d, n0, nu, true);
}

// R_y = compress(T_y R_{y+1}; D, sweeps).  Returns the tensors of R_y (unit norm) and log of the norm removed.
std::vector<MpsTensor> compress(Ctx& cx, int y, const std::vector<MpsTensor>& Aold, int D, int sweeps,
                                double* lognorm) {
  tn_handle* h = cx.h;
  std::vector<PosInfo> pos = row_positions(h, y);
  const int n = (int)pos.size();
  const bool exact = D <= 0;
  // ---- C-1: left-canonicalise a working copy of R_{y+1}
  std::vector<MpsTensor> A(n);
  for (int j = 0; j < n; j++) {
    A[j] = new_tensor(h, Aold[j].dl, Aold[j].p, Aold[j].dr);
    TN_CUDA(cudaMemcpyAsync(A[j].d, Aold[j].d, sizeof(double) * A[j].dl * A[j].p * A[j].dr, cudaMemcpyDeviceToDevice,
                            h->stream));
  }
  DBuf<double> rlast(h, 1);
  left_canonicalize(cx, A, rlast.p);
  // ---- static bond dimensions of the new MPS (zero-padded where the numerical rank is lower)
  std::vector<int> chi(n + 1, 1);
  const bool two_step = !exact && h->two_step;
  const int cap = exact ? h->exact_cap : (two_step ? 2 * D : D);   // bond kept by the zipper and the passes
  for (int j = n - 1; j >= 0; j--) {
    i64 mm = (i64)A[j].dl * pos[j].wl, nn = (i64)pos[j].pu * chi[j + 1];
    i64 full = std::min(mm, nn);
    if (exact && full > cap)
      tn_throw(TN_ERR_ARG, "exact contraction (D <= 0) needs bond %lld > TN_OPT_EXACT_CAP = %d at row %d position %d",
               (long long)full, cap, y, j);
    chi[j] = (int)std::min<i64>(cap, full);
  }
  std::vector<double*> Renv(n, nullptr), Lenv(n, nullptr);
  std::vector<MpsTensor> N(n);
  // log-scales removed from the environments: lsR[j] = ls[j], lsL[j] = ls[n + j], ls0 = ls[2n] (reading S19)
  DBuf<double> lsbuf(h, 2 * (size_t)n + 2);
  double* ls = lsbuf.p;
  TN_CUDA(cudaMemsetAsync(ls, 0, sizeof(double) * (2 * (size_t)n + 2), h->stream));
  double* d_sig0 = cx.d_scal + 1;
  double* d_safe = cx.d_scal + 2;
  double* d_dummy = cx.d_scal + 3;
  // ---- one-site variational steps (C-4; Fig. 8(d)): update the centre at q from both environments, move it on
  auto step_right = [&](int q, bool move, bool track_ls) {     // centre q -> q + 1 (left environment extended)
    const int g = chi[q], s2 = chi[q + 1];
    ThetaOp op = build_op(cx, pos[q], true, A[q], Lenv[q], g);
    DBuf<double> Z(h, (size_t)op.n * s2);
    apply_T(cx, op, Renv[q], Z.p, s2);
    if (move) {
      cx.tic(&h->st.ms_orth_svd);
      orth_columns(h, Z.p, op.n, s2, 5);
      cx.toc();
      if (Lenv[q + 1]) h->dfree(Lenv[q + 1]);
      Lenv[q + 1] = h->dalloc<double>((size_t)op.m * s2);
      apply_N(cx, op, Z.p, Lenv[q + 1], s2);
      frob_norm(h, Lenv[q + 1], op.m * s2, d_sig0);
      k_ls_step<<<1, 32, 0, h->stream>>>(d_sig0, track_ls ? ls + n + q : nullptr, track_ls ? ls + n + q + 1 : d_dummy, d_safe);
      TN_LAUNCH_CHECK(h);
      scale_by(h, Lenv[q + 1], op.m * s2, d_safe, true);
    }
    permute3(h, N[q].d, Z.p, g, pos[q].pu, s2, s2, (i64)g * s2, 1);
    free_op(cx, op);
  };
  auto step_left = [&](int q, bool move) {                     // centre q -> q - 1 (right environment extended)
    const int g = chi[q + 1], s2 = chi[q];
    ThetaOp op = build_op(cx, pos[q], false, A[q], Renv[q], g);
    DBuf<double> Z(h, (size_t)op.n * s2);
    apply_T(cx, op, Lenv[q], Z.p, s2);
    if (move) {
      cx.tic(&h->st.ms_orth_svd);
      orth_columns(h, Z.p, op.n, s2, 5);
      cx.toc();
      h->dfree(Renv[q - 1]);
      Renv[q - 1] = h->dalloc<double>((size_t)op.m * s2);
      apply_N(cx, op, Z.p, Renv[q - 1], s2);
      frob_norm(h, Renv[q - 1], op.m * s2, d_sig0);
      k_ls_step<<<1, 32, 0, h->stream>>>(d_sig0, ls + q, ls + q - 1, d_safe);
      TN_LAUNCH_CHECK(h);
      scale_by(h, Renv[q - 1], op.m * s2, d_safe, true);
    }
    permute3(h, N[q].d, Z.p, s2, pos[q].pu, g, 1, (i64)g * s2, s2);
    free_op(cx, op);
  };
  // ---- C-2/C-3: zipper right -> left
  const bool interleaved = !exact && h->schedule == 1 && h->sweep_range > 0 && n > 1;
  bool centre_swept = false;   // the centre tensor N[0] came out of a variational step (its scale sits in lsR[0] + lsL[0])
  Renv[n - 1] = h->dalloc<double>(1);
  TN_CUDA(cudaMemcpyAsync(Renv[n - 1], rlast.p, sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
  for (int j = n - 1; j >= 0; j--) {
    const int g = chi[j + 1];
    ThetaOp op = build_op(cx, pos[j], false, A[j], Renv[j], g);
    const i64 mn = std::min(op.m, op.n);
    const int ks = exact ? (int)mn : (int)std::min<i64>((i64)chi[j] + h->oversample, mn);
    DBuf<double> Vz(h, (size_t)op.n * chi[j]);
    double* C = h->dalloc<double>((size_t)op.m * chi[j]);
    if (!exact && h->svd_mode == 1 && mn > cap) svd_rand(cx, op, chi[j], ks, pos[j].pu, g, Vz.p, C, d_sig0);
    else if (h->svd_direct && svd_direct_fits(op.m, op.n)) svd_direct(cx, op, chi[j], Vz.p, C, d_sig0);
    else svd_trunc(cx, op, chi[j], ks, Vz.p, C, d_sig0);
    N[j] = new_tensor(h, chi[j], pos[j].pu, g);
    permute3(h, N[j].d, Vz.p, chi[j], pos[j].pu, g, 1, (i64)g * chi[j], chi[j]);
    // connector <- connector / sigma_1, log sigma_1 carried beside it
    k_ls_step<<<1, 32, 0, h->stream>>>(d_sig0, ls + j, j > 0 ? ls + j - 1 : ls + 2 * n, d_safe);
    TN_LAUNCH_CHECK(h);
    scale_by(h, C, op.m * chi[j], d_safe, true);
    if (j > 0) {
      Renv[j - 1] = C;
    } else {
      scale_by(h, N[0].d, (i64)N[0].dl * N[0].p * N[0].dr, C, false);
      h->dfree(C);
    }
    free_op(cx, op);
    if (interleaved && j < n - 1) {
      // ---- variational sweep of the instantaneous stage of the zipper over positions j .. kmax and
      // back.  The block [connector . N_j ... N_{n-1}] approximates (A_j W_j) ... (A_{n-1} W_{n-1}) with its left legs
      // (old bond, MPO bond) open; an orthonormal basis of the connector's range on those legs is the left
      // environment of position j (reading S21): the connector already has the environment layout.
      const int kmax = std::min(n - 1, j + h->sweep_range);
      if (Lenv[j]) h->dfree(Lenv[j]);
      if (j > 0) {
        const i64 mc = (i64)A[j].dl * pos[j].wl;
        Lenv[j] = h->dalloc<double>((size_t)mc * chi[j]);
        TN_CUDA(cudaMemcpyAsync(Lenv[j], Renv[j - 1], sizeof(double) * mc * chi[j], cudaMemcpyDeviceToDevice, h->stream));
        cx.tic(&h->st.ms_orth_svd);
        orth_columns(h, Lenv[j], mc, chi[j], 5);
        cx.toc();
      } else {
        Lenv[0] = h->dalloc<double>(1);
        fill_value(h, Lenv[0], 1, 1.0);
      }
      for (int q = j; q < kmax; q++) step_right(q, true, false);
      for (int q = kmax; q >= j; q--) step_left(q, q > 0);
      if (j == 0) centre_swept = true;
    }
  }
  // ---- C-4: one-site variational passes, alternating, first left -> right
  int centre = 0;
  if (!exact && sweeps > 0) {
    if (Lenv[0]) h->dfree(Lenv[0]);
    Lenv[0] = h->dalloc<double>(1);
    fill_value(h, Lenv[0], 1, 1.0);
    TN_CUDA(cudaMemsetAsync(ls + n, 0, sizeof(double) * n, h->stream));
    for (int sw = 0; sw < sweeps; sw++) {
      if (sw % 2 == 0) {
        for (int j = 0; j < n; j++) step_right(j, j + 1 < n, true);
        centre = n - 1;
      } else {
        for (int j = n - 1; j >= 0; j--) step_left(j, j > 0);
        centre = 0;
      }
    }
    centre_swept = true;
  }
  // ---- norm of the centre tensor -> log-scale
  const i64 nc = (i64)N[centre].dl * N[centre].p * N[centre].dr;
  frob_norm(h, N[centre].d, nc, cx.d_scal);
  scale_by(h, N[centre].d, nc, cx.d_scal, true);
  if (two_step) truncate_mps(cx, N, D, d_dummy);   // 2 chi -> chi; the norm left after the cut joins the log-scale
  else fill_value(h, d_dummy, 1, 1.0);
  double nrm = 0.0, nu = 1.0;
  std::vector<double> lsh(2 * (size_t)n + 2);
  TN_CUDA(cudaMemcpyAsync(&nrm, cx.d_scal, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaMemcpyAsync(&nu, d_dummy, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaMemcpyAsync(lsh.data(), ls, sizeof(double) * lsh.size(), cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaStreamSynchronize(h->stream));
  if (!(nrm > 0.0) || !std::isfinite(nrm) || !(nu > 0.0) || !std::isfinite(nu))
    tn_throw(TN_ERR_NUMERIC, "row %d: boundary MPS norm is %g (after the 2 chi -> chi cut: %g)", y, nrm, nu);
  *lognorm = std::log(nrm) + std::log(nu) + (centre_swept ? lsh[centre] + lsh[n + centre] : lsh[2 * (size_t)n]);
  if (!std::isfinite(*lognorm)) tn_throw(TN_ERR_NUMERIC, "row %d: log-norm is not finite", y);
  for (int j = 0; j < n; j++) {
    h->dfree(A[j].d);
    if (Renv[j]) h->dfree(Renv[j]);
    if (Lenv[j]) h->dfree(Lenv[j]);
  }
  return N;
}

}  // namespace

void mps_free(tn_handle* h) {
  for (auto& row : h->rows)
    for (auto& t : row)
      if (t.d) h->dfree(t.d);
  h->rows.clear();
  h->lognorm.clear();
  h->have_mps = false;
  h->have_logz = false;
}

void contract_run(tn_handle* h, int D, int sweeps) {
  mps_free(h);
  h->svd_skip_first = 0;
  Ctx cx;
  cx.h = h;
  DBuf<int> ints(h, 4);
  DBuf<double> dbl(h, 8);
  cx.d_keep = ints.p; cx.d_flag = ints.p + 1;
  cx.d_stat = dbl.p; cx.d_scal = dbl.p + 4;
  TN_CUDA(cudaMemsetAsync(dbl.p, 0, sizeof(double) * 8, h->stream));
  cudaEvent_t e0, e1;
  TN_CUDA(cudaEventCreate(&e0)); TN_CUDA(cudaEventCreate(&e1));
  TN_CUDA(cudaEventRecord(e0, h->stream));
  const int Ly = h->Ly;
  const int npos = h->has_med() ? 2 * h->Lx - 1 : h->Lx;
  h->rows.assign(Ly + 1, std::vector<MpsTensor>());
  h->lognorm.assign(Ly + 1, 0.0);
  h->rows[Ly].resize(npos);
  for (int j = 0; j < npos; j++) {
    h->rows[Ly][j] = new_tensor(h, 1, 1, 1);
    fill_value(h, h->rows[Ly][j].d, 1, 1.0);
  }
  try {
    for (int y = Ly - 1; y >= 1; y--) {
      h->rows[y] = compress(cx, y, h->rows[y + 1], D, sweeps, &h->lognorm[y]);
      h->st.rows_contracted++;
      cx.flush();
    }
  } catch (...) {
    cx.flush();
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    throw;
  }
  double stat = 0.0;
  TN_CUDA(cudaMemcpyAsync(&stat, cx.d_stat, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaEventRecord(e1, h->stream));
  TN_CUDA(cudaStreamSynchronize(h->stream));
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  h->st.ms_contract += ms;
  h->st.min_sigma_rel = std::max(h->st.min_sigma_rel, stat);
  h->D = D; h->sweeps = sweeps;
  h->have_mps = true;
}
