// Launchers of the shared device kernels (kernels.cu).  All work goes to h->stream.
#pragma once
#include "tn_common.cuh"
#include "gemm.cuh"

#define TN_LAUNCH_CHECK(h)                                                              \
  do {                                                                                  \
    (h)->st.kernel_launches++;                                                          \
    cudaError_t e__ = cudaPeekAtLastError();                                            \
    if (e__ != cudaSuccess) tn_throw(TN_ERR_CUDA, "launch failed: %s (%s:%d)",          \
                                     cudaGetErrorString(e__), __FILE__, __LINE__);     \
  } while (0)

static inline int cdiv(i64 a, i64 b) { return (int)((a + b - 1) / b); }

// X[i] = uniform(-1,1) from a counter-based hash of (seed, i)
void fill_random(tn_handle* h, double* X, i64 n, uint64_t seed);
void fill_value(tn_handle* h, double* X, i64 n, double v);
// X[(p', gamma)][col], p' < pu, gamma < g (<= 4096), col < ks (<= 1024): counter-based, layout-free (randomized SVD)
void fill_random_pgc(tn_handle* h, double* X, int pu, int g, int ks, uint64_t seed);
// out[i0][i1][i2] = in[i0*s0 + i1*s1 + i2*s2]; entries whose index along `mask_axis` (0..2, -1 = none)
// is >= *keep (device int) are written as exact zeros.
void permute3(tn_handle* h, double* out, const double* in, int n0, int n1, int n2, i64 s0, i64 s1, i64 s2,
              int mask_axis = -1, const int* keep = nullptr);
// X *= *s (device scalar) or X *= 1 / *s
void scale_by(tn_handle* h, double* X, i64 n, const double* s, bool inverse);
// *out = ||X||_F  (deterministic two-stage reduction)
void frob_norm(tn_handle* h, const double* X, i64 n, double* out);

// One-sided Jacobi on the ROWS of Min [c x r] (ld): finds orthogonal W with rows of W^T Min mutually
// orthogonal.  Outputs sorted by descending row norm: Mout = W^T Min [c x r], Wt = W^T [c x c], sig [c].
void jacobi_rows(tn_handle* h, const double* Min, int ld, int c, int r, double* Mout, double* Wt, double* sig);

// Orthonormalise the columns of Y [m x k] (ld = k) in place (orth.cu): up to `passes` rounds of pivot-floored
// Cholesky-QR (k <= 96; Gram -> Jacobi eigen-decomposition rounds above that), early exit once Y^T Y = I to
// rounding; rank-deficient / exactly-zero columns are harmless (reading S6).
void orth_columns(tn_handle* h, double* Y, i64 m, int k, int passes);

// ---- projector / fold maps on arrays laid out [outer][index][s] ----------
// bond -> state space of the LEFT leg of a site:   fold:  Yk[o][a][s]      = sum_r BhS[r][a] Y[o][r][s]
//                                                  else:  Yk[o][(a,cl)][s] = sum_ch wC[cl][ch] Y[o][(Pl a, Pi ch)][s]
void map_L(tn_handle* h, const CellDev& c, bool fold, const double* Y, double* Yk, int outer, int s);
void map_LT(tn_handle* h, const CellDev& c, bool fold, const double* Yk, double* Y, int outer, int s);
// bond -> state space of the RIGHT leg: Yk[o][(a,cl)][s] = Y[o][(Pr a, Po cl)][s]  and its transpose (scatter-sum)
void map_R(tn_handle* h, const CellDev& c, const double* Y, double* Yk, int outer, int s);
void map_RT(tn_handle* h, const CellDev& c, const double* Yk, double* Y, int outer, int s);

// Theta-core of a site (Fig. 7(a,b) PAPER.md:155-161):
//   Tc[(x,k),(b,g)] = g(k,b) * sum_y A[x][Pd b][y] * Ek[(y,k)][g],  A: [dx][pd][dy] row-major
void theta_core(tn_handle* h, const CellDev& c, const double* A, int dx, int dy, const double* Ek, int g,
                double* Tc);
// mediating tensor pieces (Fig. 7(c,d) PAPER.md:163)
//   Theta[(al,r,o),(q',g)] = sum_i' Bd[q',i'] T1[(al,o),(r,i',g)]
void med_apply_bd(tn_handle* h, const double* T1, const double* Bd, double* Theta, int al, int n_o, int n_r,
                  int n_i, int n_q, int g);
//   ThetaL[(ar,l',i'),(q',g)] = TL[(ar,l'),g] * Bd[q',i']
void med_outer_bd(tn_handle* h, const double* TL, const double* Bd, double* Theta, i64 rows, int n_i, int n_q,
                  int g);
