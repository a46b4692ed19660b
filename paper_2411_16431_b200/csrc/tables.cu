// a1: local tables.  Clustered (Potts) form of the Ising instance, Eq. (3); projectors
// and compressed edge energies, Eqs. (4)-(5) PAPER.md:76-84, Fig. 2; Boltzmann bond
// tensors exp(-beta Ebar), Fig. 5(c) PAPER.md:133.  One CTA per cell enumerates the 2^n_s states of each
// sub-cluster, the 2^(n_s/2) x 2^(n_s/2) inter-sub-cluster tables and the projected edge matrices.
#include "kernels.cuh"

struct CellEdge {
  int type;   // 0..2 intra sub s | 3,4 chain s->s+1 | 5 horizontal-in | 6 vertical-in | 7 diagonal-in | 8 field
  int pu, pv; // bit positions (see tables_create)
  double J;
};
struct CellBuild {   // per-cell build descriptor (device)
  int S, ns, half;
  int m_right_left;  // m_right of the left neighbour   (0 if none)
  int m_down_up;     // m_down of the upper neighbour
  int m_dout_ul;     // m_dout of the upper-left neighbour
  int m_up, m_down;  // this cell's vertical masks (bits of the vertical sub-cluster)
  // mutable outputs (device pointers, non-const views of CellDev's)
  double *wA, *X, *Yc, *wC, *Bh, *Bv, *Bd, *BhS, *BvS;
  int *Pl, *Pr, *Pu, *Pd, *Pi, *Po;
};

__device__ __forceinline__ double sgn_bit(int state, int bit) { return 1.0 - 2.0 * ((state >> bit) & 1); }
__device__ __forceinline__ int pext8(int v, int mask) {
  int out = 0, bit = 0;
  for (int i = 0; i < 8; i++)
    if ((mask >> i) & 1) { out |= ((v >> i) & 1) << bit; bit++; }
  return out;
}
__device__ __forceinline__ int rank_in(int mask, int bit) { return __popc(mask & ((1 << bit) - 1)); }

__device__ double block_min(double v, double* sh) {
  int tid = threadIdx.x;
  sh[tid] = v;
  __syncthreads();
  for (int o = blockDim.x / 2; o > 0; o >>= 1) {
    if (tid < o) sh[tid] = fmin(sh[tid], sh[tid + o]);
    __syncthreads();
  }
  double r = sh[0];
  __syncthreads();
  return r;
}

__global__ void __launch_bounds__(256) k_tables(const CellDev* cells, const CellBuild* builds, const CellEdge* edges,
                                                const int* eptr, double beta, double* offsets) {
  __shared__ double sE[256], sh[256], sT[256], sW[256];
  const int cell = blockIdx.x, tid = threadIdx.x;
  const CellDev c = cells[cell];
  const CellBuild B = builds[cell];
  const CellEdge* E = edges + eptr[cell];
  const int ne = eptr[cell + 1] - eptr[cell];
  const int half = B.half, nH = 1 << half;
  double off = 0.0;

  // ---- sub-cluster 0: wA
  {
    double e = 0.0;
    if (tid < c.nA)
      for (int i = 0; i < ne; i++) {
        if (E[i].type == 0) e += E[i].J * sgn_bit(tid, E[i].pu) * sgn_bit(tid, E[i].pv);
        else if (E[i].type == 8 && E[i].pu == 0) e += E[i].J * sgn_bit(tid, E[i].pv);
      }
    double mn = block_min(tid < c.nA ? e : INFINITY, sh);
    if (tid < c.nA) B.wA[tid] = exp(-beta * (e - mn));
    off += mn;
  }
  // ---- sub-cluster 1 and the A-B table: X[t][b] = wAB[t][b_lo] * wB[b]   (S == 1: identity)
  if (B.S >= 2) {
    double e = 0.0;
    if (tid < c.nB)
      for (int i = 0; i < ne; i++) {
        if (E[i].type == 1) e += E[i].J * sgn_bit(tid, E[i].pu) * sgn_bit(tid, E[i].pv);
        else if (E[i].type == 8 && E[i].pu == 1) e += E[i].J * sgn_bit(tid, E[i].pv);
      }
    double mn = block_min(tid < c.nB ? e : INFINITY, sh);
    if (tid < c.nB) sW[tid] = exp(-beta * (e - mn));   // wB
    off += mn;
    double e2 = 0.0;
    if (tid < nH * nH) {
      int t = tid / nH, bl = tid % nH;
      for (int i = 0; i < ne; i++)
        if (E[i].type == 3) e2 += E[i].J * sgn_bit(t, E[i].pu) * sgn_bit(bl, E[i].pv);
    }
    double mn2 = block_min(tid < nH * nH ? e2 : INFINITY, sh);
    if (tid < nH * nH) sT[tid] = exp(-beta * (e2 - mn2));   // wAB[t][b_lo]
    off += mn2;
    __syncthreads();
    for (int i = tid; i < c.nT * c.nB; i += blockDim.x) {
      int t = i / c.nB, b = i % c.nB;
      B.X[i] = sT[t * nH + (b & (nH - 1))] * sW[b];
    }
    __syncthreads();
  } else {
    for (int i = tid; i < c.nT * c.nB; i += blockDim.x) B.X[i] = (i / c.nB == i % c.nB) ? 1.0 : 0.0;
  }
  // ---- sub-cluster 2: wC[cl][ch], Yc[b][cl] = wBC[b_hi][cl]
  if (B.S == 3) {
    double e = 0.0;
    if (tid < c.nA)
      for (int i = 0; i < ne; i++) {
        if (E[i].type == 2) e += E[i].J * sgn_bit(tid, E[i].pu) * sgn_bit(tid, E[i].pv);
        else if (E[i].type == 8 && E[i].pu == 2) e += E[i].J * sgn_bit(tid, E[i].pv);
      }
    double mn = block_min(tid < c.nA ? e : INFINITY, sh);
    if (tid < c.nA) B.wC[(tid & (nH - 1)) * c.nCh + (tid >> half)] = exp(-beta * (e - mn));
    off += mn;
    double e2 = 0.0;
    if (tid < nH * nH) {
      int bh = tid / nH, cl = tid % nH;
      for (int i = 0; i < ne; i++)
        if (E[i].type == 4) e2 += E[i].J * sgn_bit(bh, E[i].pu) * sgn_bit(cl, E[i].pv);
    }
    double mn2 = block_min(tid < nH * nH ? e2 : INFINITY, sh);
    if (tid < nH * nH) sT[tid] = exp(-beta * (e2 - mn2));
    off += mn2;
    __syncthreads();
    for (int i = tid; i < c.nB * c.nCl; i += blockDim.x) {
      int b = i / c.nCl, cl = i % c.nCl;
      B.Yc[i] = sT[(b >> half) * nH + cl];
    }
    __syncthreads();
  } else {
    for (int i = tid; i < c.nB * c.nCl; i += blockDim.x) B.Yc[i] = 1.0;
    if (tid == 0) B.wC[0] = 1.0;
  }
  // ---- projector index tables, Eq. (5): bits of the coupled spins packed in increasing order
  if (tid < c.nA) {
    B.Pl[tid] = pext8(tid, c.m_left);
    B.Pr[tid] = pext8(tid, c.m_right);
  }
  if (tid < c.nB) {
    B.Pu[tid] = pext8(tid, B.m_up);
    B.Pd[tid] = pext8(tid, B.m_down);
  }
  if (tid < c.nCh) B.Pi[tid] = pext8(tid, c.m_din);
  if (tid < c.nCl) B.Po[tid] = pext8(tid, c.m_dout);
  __syncthreads();
  // ---- edge matrices (bond tensors): Bh [bh_rows x n_l], Bv [bv_rows x n_u], Bd [bd_rows x n_i]
  for (int kind = 0; kind < 3; kind++) {
    const int type = 5 + kind;
    const int rows = kind == 0 ? c.bh_rows : kind == 1 ? c.bv_rows : c.bd_rows;
    const int cols = kind == 0 ? c.n_l : kind == 1 ? c.n_u : c.n_i;
    const int mrow = kind == 0 ? B.m_right_left : kind == 1 ? B.m_down_up : B.m_dout_ul;
    const int mcol = kind == 0 ? c.m_left : kind == 1 ? B.m_up : c.m_din;
    double* out = kind == 0 ? B.Bh : kind == 1 ? B.Bv : B.Bd;
    double mn = INFINITY;
    for (int i = tid; i < rows * cols; i += blockDim.x) {
      int r = i / cols, l = i % cols;
      double e = 0.0;
      for (int q = 0; q < ne; q++)
        if (E[q].type == type) {
          int pv = kind == 2 ? E[q].pv - half : E[q].pv;
          e += E[q].J * sgn_bit(r, rank_in(mrow, E[q].pu)) * sgn_bit(l, rank_in(mcol, pv));
        }
      out[i] = e;
      mn = fmin(mn, e);
    }
    mn = block_min(mn, sh);
    for (int i = tid; i < rows * cols; i += blockDim.x) out[i] = exp(-beta * (out[i] - mn));
    off += mn;
    __syncthreads();
  }
  for (int i = tid; i < c.bh_rows * c.nA; i += blockDim.x) B.BhS[i] = B.Bh[(i / c.nA) * c.n_l + B.Pl[i % c.nA]];
  for (int i = tid; i < c.bv_rows * c.nB; i += blockDim.x) B.BvS[i] = B.Bv[(i / c.nB) * c.n_u + B.Pu[i % c.nB]];
  if (tid == 0) offsets[cell] = off;
}

// ---------------------------------------------------------------------------------------------
static int popc(int v) { return __builtin_popcount((unsigned)v); }

void tables_create(tn_handle* h) {
  const int Ly = h->Ly, Lx = h->Lx, S = h->S, ns = h->ns, half = ns / 2;
  const int ncell = Ly * Lx, vsub = std::min(1, S - 1);
  const int nA = 1 << ns, nH = 1 << half;
  std::vector<std::vector<CellEdge>> ce(ncell);
  struct Masks { int left = 0, right = 0, up = 0, down = 0, din = 0, dout = 0; };
  std::vector<Masks> mk(ncell);
  std::vector<int> sub_of(h->n_spins), pos_of(h->n_spins);
  for (int i = 0; i < h->n_spins; i++) { sub_of[i] = h->bit_of[i] / ns; pos_of[i] = h->bit_of[i] % ns; }
  for (i64 e = 0; e < h->n_edges; e++) {
    int u = h->edge_u[e], v = h->edge_v[e];
    double J = h->J[e];
    if (u == v) tn_throw(TN_ERR_GEOMETRY, "edge %lld is a self-loop on spin %d", (long long)e, u);
    int cu = h->cell_of[u], cv = h->cell_of[v];
    if (cu == cv) {
      int su = sub_of[u], sv = sub_of[v], pu = pos_of[u], pv = pos_of[v];
      if (su == sv) { ce[cu].push_back({su, pu, pv, J}); continue; }
      if (su > sv) { std::swap(su, sv); std::swap(pu, pv); std::swap(u, v); }
      if (sv != su + 1 || pu < half || pv >= half)
        tn_throw(TN_ERR_GEOMETRY, "edge %lld (spins %d,%d): intra-cell edges must stay inside a sub-cluster or join "
                 "the hi half of sub-cluster s to the lo half of s+1", (long long)e, h->edge_u[e], h->edge_v[e]);
      ce[cu].push_back({3 + su, pu - half, pv, J});
      continue;
    }
    if (cv < cu) { std::swap(u, v); std::swap(cu, cv); }
    int yu = cu / Lx, xu = cu % Lx, yv = cv / Lx, xv = cv % Lx;
    int su = sub_of[u], sv = sub_of[v], pu = pos_of[u], pv = pos_of[v];
    if (yv == yu && xv == xu + 1) {
      if (su != 0 || sv != 0)
        tn_throw(TN_ERR_GEOMETRY, "edge %lld (spins %d,%d): horizontal edges must join sub-cluster 0 to sub-cluster 0",
                 (long long)e, h->edge_u[e], h->edge_v[e]);
      mk[cu].right |= 1 << pu; mk[cv].left |= 1 << pv;
      ce[cv].push_back({5, pu, pv, J});
    } else if (yv == yu + 1 && xv == xu) {
      if (su != vsub || sv != vsub)
        tn_throw(TN_ERR_GEOMETRY, "edge %lld (spins %d,%d): vertical edges must join sub-cluster %d to sub-cluster %d",
                 (long long)e, h->edge_u[e], h->edge_v[e], vsub, vsub);
      mk[cu].down |= 1 << pu; mk[cv].up |= 1 << pv;
      ce[cv].push_back({6, pu, pv, J});
    } else if (yv == yu + 1 && xv == xu + 1) {
      if (S != 3 || su != 2 || sv != 2 || pu >= half || pv < half)
        tn_throw(TN_ERR_GEOMETRY, "edge %lld (spins %d,%d): diagonal edges must join the lo half of sub-cluster 2 of "
                 "(x,y) to the hi half of sub-cluster 2 of (x+1,y+1)", (long long)e, h->edge_u[e], h->edge_v[e]);
      mk[cu].dout |= 1 << pu; mk[cv].din |= 1 << (pv - half);
      ce[cv].push_back({7, pu, pv, J});
    } else {
      tn_throw(TN_ERR_GEOMETRY, "edge %lld (spins %d,%d) joins cells (%d,%d) and (%d,%d): only nearest neighbours and "
               "the (x+1,y+1) diagonal are allowed", (long long)e, h->edge_u[e], h->edge_v[e], yu, xu, yv, xv);
    }
  }
  for (int i = 0; i < h->n_spins; i++)
    if (h->h[i] != 0.0) ce[h->cell_of[i]].push_back({8, sub_of[i], pos_of[i], h->h[i]});

  // descriptors and pool layout
  h->cells.assign(ncell, CellDev());
  std::vector<CellBuild> builds(ncell);
  size_t nd = 0, ni = 0;
  auto takeD = [&](size_t n) { size_t o = nd; nd += (n + 1) & ~(size_t)1; return o; };
  auto takeI = [&](size_t n) { size_t o = ni; ni += (n + 3) & ~(size_t)3; return o; };
  std::vector<size_t> od(ncell * 9), oi(ncell * 6);
  for (int cidx = 0; cidx < ncell; cidx++) {
    int y = cidx / Lx, x = cidx % Lx;
    CellDev& c = h->cells[cidx];
    const Masks& m = mk[cidx];
    c.nA = nA;
    c.nB = nA;
    c.nCl = S == 3 ? nH : 1;
    c.nCh = S == 3 ? nH : 1;
    c.nK = c.nA * c.nCl;
    c.tshift = S == 1 ? 0 : half;
    c.nT = S == 1 ? nA : nH;
    c.m_left = m.left; c.m_right = m.right; c.m_din = m.din; c.m_dout = m.dout;
    c.m_up = m.up; c.m_down = m.down;
    c.n_l = 1 << popc(m.left); c.n_r = 1 << popc(m.right);
    c.n_u = 1 << popc(m.up); c.n_d = 1 << popc(m.down);
    c.n_i = 1 << popc(m.din); c.n_o = 1 << popc(m.dout);
    c.bh_rows = x > 0 ? 1 << popc(mk[cidx - 1].right) : 1;
    c.bv_rows = y > 0 ? 1 << popc(mk[cidx - Lx].down) : 1;
    c.bd_rows = (x > 0 && y > 0) ? 1 << popc(mk[cidx - Lx - 1].dout) : 1;
    CellBuild& b = builds[cidx];
    b.S = S; b.ns = ns; b.half = half;
    b.m_right_left = x > 0 ? mk[cidx - 1].right : 0;
    b.m_down_up = y > 0 ? mk[cidx - Lx].down : 0;
    b.m_dout_ul = (x > 0 && y > 0) ? mk[cidx - Lx - 1].dout : 0;
    b.m_up = m.up; b.m_down = m.down;
    size_t* o = &od[cidx * 9];
    o[0] = takeD(c.nA); o[1] = takeD((size_t)c.nT * c.nB); o[2] = takeD((size_t)c.nB * c.nCl);
    o[3] = takeD((size_t)c.nCl * c.nCh); o[4] = takeD((size_t)c.bh_rows * c.n_l);
    o[5] = takeD((size_t)c.bv_rows * c.n_u); o[6] = takeD((size_t)c.bd_rows * c.n_i);
    o[7] = takeD((size_t)c.bh_rows * c.nA); o[8] = takeD((size_t)c.bv_rows * c.nB);
    size_t* q = &oi[cidx * 6];
    q[0] = takeI(c.nA); q[1] = takeI(c.nA); q[2] = takeI(c.nB); q[3] = takeI(c.nB); q[4] = takeI(c.nCh); q[5] = takeI(c.nCl);
  }
  h->pool_d = h->dalloc<double>(nd);
  h->pool_i = h->dalloc<int>(ni);
  for (int cidx = 0; cidx < ncell; cidx++) {
    CellDev& c = h->cells[cidx];
    CellBuild& b = builds[cidx];
    size_t* o = &od[cidx * 9];
    size_t* q = &oi[cidx * 6];
    b.wA = h->pool_d + o[0]; b.X = h->pool_d + o[1]; b.Yc = h->pool_d + o[2]; b.wC = h->pool_d + o[3];
    b.Bh = h->pool_d + o[4]; b.Bv = h->pool_d + o[5]; b.Bd = h->pool_d + o[6];
    b.BhS = h->pool_d + o[7]; b.BvS = h->pool_d + o[8];
    b.Pl = h->pool_i + q[0]; b.Pr = h->pool_i + q[1]; b.Pu = h->pool_i + q[2]; b.Pd = h->pool_i + q[3];
    b.Pi = h->pool_i + q[4]; b.Po = h->pool_i + q[5];
    c.wA = b.wA; c.X = b.X; c.Yc = b.Yc; c.wC = b.wC; c.Bh = b.Bh; c.Bv = b.Bv; c.Bd = b.Bd;
    c.BhS = b.BhS; c.BvS = b.BvS;
    c.Pl = b.Pl; c.Pr = b.Pr; c.Pu = b.Pu; c.Pd = b.Pd; c.Pi = b.Pi; c.Po = b.Po;
  }
  std::vector<int> eptr(ncell + 1, 0);
  std::vector<CellEdge> flat;
  for (int cidx = 0; cidx < ncell; cidx++) {
    flat.insert(flat.end(), ce[cidx].begin(), ce[cidx].end());
    eptr[cidx + 1] = (int)flat.size();
  }
  h->d_cells = h->dalloc<CellDev>(ncell);
  h->d_cell_desc = h->dalloc<CellBuild>(ncell);
  h->d_cell_edges = h->dalloc<CellEdge>(flat.size() + 1);
  h->d_cell_edge_ptr = h->dalloc<int>(ncell + 1);
  h->d_offsets = h->dalloc<double>(ncell);
  TN_CUDA(cudaMemcpy(h->d_cells, h->cells.data(), sizeof(CellDev) * ncell, cudaMemcpyHostToDevice));
  TN_CUDA(cudaMemcpy(h->d_cell_desc, builds.data(), sizeof(CellBuild) * ncell, cudaMemcpyHostToDevice));
  if (!flat.empty())
    TN_CUDA(cudaMemcpy(h->d_cell_edges, flat.data(), sizeof(CellEdge) * flat.size(), cudaMemcpyHostToDevice));
  TN_CUDA(cudaMemcpy(h->d_cell_edge_ptr, eptr.data(), sizeof(int) * (ncell + 1), cudaMemcpyHostToDevice));
}

void tables_set_beta(tn_handle* h, double beta) {
  const int ncell = h->Ly * h->Lx;
  {
    StageTimer t(h, &h->st.ms_tables);
    k_tables<<<ncell, 256, 0, h->stream>>>(h->d_cells, (const CellBuild*)h->d_cell_desc,
                                           (const CellEdge*)h->d_cell_edges, h->d_cell_edge_ptr, beta, h->d_offsets);
    TN_LAUNCH_CHECK(h);
  }
  std::vector<double> off(ncell);
  TN_CUDA(cudaMemcpyAsync(off.data(), h->d_offsets, sizeof(double) * ncell, cudaMemcpyDeviceToHost, h->stream));
  TN_CUDA(cudaStreamSynchronize(h->stream));
  double s = 0.0;
  for (int i = 0; i < ncell; i++) s += off[i];
  if (!std::isfinite(s)) tn_throw(TN_ERR_NUMERIC, "non-finite table offset");
  h->offset = s;
  h->beta = beta;
}

void tables_destroy(tn_handle* h) {
  for (void* p : {(void*)h->pool_d, (void*)h->pool_i, (void*)h->d_cells, h->d_cell_desc, h->d_cell_edges,
                  (void*)h->d_cell_edge_ptr, (void*)h->d_offsets})
    if (p) h->dfree(p);
  h->pool_d = nullptr; h->pool_i = nullptr; h->d_cells = nullptr; h->d_cell_desc = nullptr;
  h->d_cell_edges = nullptr; h->d_cell_edge_ptr = nullptr; h->d_offsets = nullptr;
}
