// S5: from-scratch rebuild  N_sigma = A_sigma^{-1}  by a two-level blocked right-looking LU with partial pivoting,
// batched over all B*2 matrices (each with its own order k).  BASELINE.json: "a batched LU-based rebuild".
//
//   F = the non-current N buffer (A, overwritten by its LU factors: P A = L U)
//   X = the current N buffer     (starts as I; becomes X' = L^-1 in position space, then N' = U^-1 X'; N = N' P)
//
// Kernels: k_lu_panel / k_lu_panel_cl (unblocked LU of a 32-column panel: one CTA, or an 8-CTA cluster per matrix),
// k_lu_swap_range, k_lu_trsm_range (inside the outer block of 128 columns), k_lu_tri_inv (explicit 128 x 128 triangular
// inverses), k_lu_copyback, k_lu_perm / k_lu_scatter_cols / k_lu_flip; the rank-32 and rank-128 updates (TDescLU2) run on
// the TMA-staged DMMA tiles of gemm_tma.cuh.  The blocking is described above kLuOuter below.
#pragma once
#include <cooperative_groups.h>

#include "gemm_dmma.cuh"
#include "gemm_tma.cuh"
#include "walker_state.cuh"

namespace ctaux {

constexpr int kLuNb = 32;

__global__ void k_lu_init_identity(DevCtx c) {
  const int w = blockIdx.y >> 1, sp = blockIdx.y & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  double* X = c.N(w, sp, st.n_cur);
  const size_t total = (size_t)k * k;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(idx % k), j = (int)(idx / k);
    X[(size_t)j * c.ld + i] = (i == j) ? 1.0 : 0.0;
  }
}

__global__ void __launch_bounds__(1024) k_lu_panel(DevCtx c, int j0, int* detsign) {
  const int w = blockIdx.x >> 1, sp = blockIdx.x & 1;
  WalkerState& st = c.ws[w];
  const int k = st.k;
  if (j0 >= k) return;
  const int j1 = (j0 + kLuNb < k) ? j0 + kLuNb : k;
  double* F = c.N(w, sp, st.n_cur ^ 1);
  int* ipiv = c.perm + ((size_t)w * 2 + sp) * c.ld;
  const int ld = c.ld, tid = threadIdx.x, nt = blockDim.x;
  __shared__ double s_val[32];
  __shared__ int s_idx[32];
  __shared__ int s_p;
  __shared__ double s_row[kLuNb];
  for (int col = j0; col < j1; ++col) {
    // pivot search in column col, rows col..k-1 (ties: smallest row index, as a serial scan would)
    double best = -1.0;
    int bi = col;
    for (int i = col + tid; i < k; i += nt) {
      const double v = fabs(F[(size_t)col * ld + i]);
      if (v > best) { best = v; bi = i; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double ov = __shfl_xor_sync(0xffffffffu, best, o);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
      if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
    }
    if ((tid & 31) == 0) { s_val[tid >> 5] = best; s_idx[tid >> 5] = bi; }
    __syncthreads();
    if (tid == 0) {
      double b = s_val[0];
      int ix = s_idx[0];
      for (int q = 1; q < (nt >> 5); ++q)
        if (s_val[q] > b || (s_val[q] == b && s_idx[q] < ix)) { b = s_val[q]; ix = s_idx[q]; }
      s_p = ix;
      ipiv[col] = ix;
      if (!(b > 0.0)) st.status = -4;  // CTAUX_ESINGULAR
      if (detsign) {
        int sg = detsign[w * 2 + sp];
        if (ix != col) sg = -sg;
        if (F[(size_t)col * ld + ix] < 0.0) sg = -sg;
        detsign[w * 2 + sp] = sg;
      }
    }
    __syncthreads();
    const int pr = s_p;
    // interchange rows col <-> pr inside the panel; publish the pivot row
    if (tid < j1 - j0) {
      const int jj = j0 + tid;
      double a = F[(size_t)jj * ld + col];
      if (pr != col) {
        const double b = F[(size_t)jj * ld + pr];
        F[(size_t)jj * ld + col] = b;
        F[(size_t)jj * ld + pr] = a;
        a = b;
      }
      s_row[tid] = a;
    }
    __syncthreads();
    const double piv = s_row[col - j0];
    if (piv != 0.0) {
      for (int i = col + 1 + tid; i < k; i += nt) {
        const double l = F[(size_t)col * ld + i] / piv;
        F[(size_t)col * ld + i] = l;
        for (int jj = col + 1; jj < j1; ++jj) F[(size_t)jj * ld + i] -= l * s_row[jj - j0];
      }
    }
    __syncthreads();
  }
}

// Panel factorisation spread over a thread-block CLUSTER of 8 CTAs per matrix (large k): the rows j0..k of the
// panel are dealt out in 8 contiguous slabs, each held in its CTA's shared memory for the whole panel, so the
// kLuNb column steps run out of shared memory instead of streaming the panel through one SM's L2 port
// (k_lu_panel: 200-600 us per panel at k = 1300-3600).  Per column: local pivot search, candidates exchanged
// through distributed shared memory (cluster barrier), pivot row broadcast + row interchange (cluster barrier),
// local elimination.  Same pivot choice as k_lu_panel (largest magnitude, smallest row index on ties).
constexpr int kLuCl = 8;
constexpr int kLuClThreads = 512;
// dynamic shared memory of k_lu_panel_cl<NB>, in doubles
__host__ __device__ inline int lu_cl_smem_doubles(int rl_cap, int nbw) {
  return rl_cap * (nbw + 1) + 2 * kLuCl * (nbw + 2) + 2 * nbw;
}

template <int NB>   // panel width (32 in use)
__global__ void __cluster_dims__(kLuCl, 1, 1) __launch_bounds__(kLuClThreads, 1)
    k_lu_panel_cl(DevCtx c, int j0, int* detsign, int rl_cap) {
  constexpr int kLuNb = NB, kLuPad = NB + 1, kLuMsg = NB + 2;   // (shadow the file-level panel width)
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  extern __shared__ __align__(16) double lsm[];
  const int prob = blockIdx.x / kLuCl, rank = (int)cluster.block_rank();
  const int w = prob >> 1, sp = prob & 1;
  WalkerState& st = c.ws[w];
  const int k = st.k;
  if (j0 >= k) return;                       // identical for all CTAs of the cluster
  const int j1 = (j0 + kLuNb < k) ? j0 + kLuNb : k;
  const int nb = j1 - j0;
  double* F = c.N(w, sp, st.n_cur ^ 1);
  int* ipiv = c.perm + ((size_t)w * 2 + sp) * c.ld;
  const int ld = c.ld, tid = threadIdx.x;
  const int rows = k - j0;
  const int R = (rows + kLuCl - 1) / kLuCl;  // rows per CTA (<= rl_cap)
  const int r0 = j0 + rank * R;              // first global row of this slab
  int nloc = k - r0; if (nloc > R) nloc = R; if (nloc < 0) nloc = 0;
  double* A = lsm;                                       // [rl_cap][kLuPad] row-major: A[i*kLuPad + cc]
  double* msg = lsm + (size_t)rl_cap * kLuPad;           // [2 parities][kLuCl senders][kLuMsg]
  double* rowc = msg + 2 * kLuCl * kLuMsg;               // [2 parities][kLuNb]  row `col` (from its owner)
  __shared__ double s_val[kLuClThreads / 32];
  __shared__ int s_idx[kLuClThreads / 32];
  __shared__ int s_best;

  for (int idx = tid; idx < nloc * nb; idx += kLuClThreads) {
    const int i = idx % nloc, cc = idx / nloc;
    A[i * kLuPad + cc] = F[(size_t)(j0 + cc) * ld + r0 + i];
  }
  // per-column exchange: every CTA sends its message (and the owner of row `col` that row) to all CTAs with st.async,
  // which completes the bytes on the RECEIVER's mbarrier -- one one-way message instead of stores + a cluster barrier
  // Two mbarriers, one per buffer parity: a fast CTA may send column cc + 1 while a slow one still waits for column cc;
  // those bytes must not be counted on the phase of column cc.  (Messages for cc + 2 reach barrier cc & 1 only after its
  // phase cc has completed everywhere: a CTA sends cc + 2 after it has received cc + 1 from all, and each of those was sent
  // after its sender had passed the wait of column cc.)
  __shared__ uint64_t cbar[2];
  if (tid == 0) { mbar_init(cbar, 1); mbar_init(cbar + 1, 1); mbar_fence_init(); }
  const uint32_t msg_a = smem_u32(msg), rowc_a = smem_u32(rowc);
  constexpr uint32_t kColBytes = (uint32_t)((kLuCl * kLuMsg + kLuNb) * 8);
  cluster.sync();

  for (int cc = 0; cc < nb; ++cc) {
    const int col = j0 + cc, par = cc & 1;
    // 1. local pivot candidate over the local rows with global index >= col
    double best = -1.0;
    int bi = 0x7fffffff;
    for (int i = tid; i < nloc; i += kLuClThreads) {
      const int gi = r0 + i;
      if (gi >= col) {
        const double v = fabs(A[i * kLuPad + cc]);
        if (v > best || (v == best && gi < bi)) { best = v; bi = gi; }
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double ov = __shfl_xor_sync(0xffffffffu, best, o);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
      if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
    }
    if ((tid & 31) == 0) { s_val[tid >> 5] = best; s_idx[tid >> 5] = bi; }
    __syncthreads();
    if (tid == 0) {
      double b = s_val[0];
      int ix = s_idx[0];
      for (int q = 1; q < kLuClThreads / 32; ++q)
        if (s_val[q] > b || (s_val[q] == b && s_idx[q] < ix)) { b = s_val[q]; ix = s_idx[q]; }
      s_val[0] = b; s_best = ix;
    }
    __syncthreads();
    // 2. ONE message per CTA to every CTA: candidate magnitude, row index and the candidate row itself; the owner
    //    of row `col` also sends that row (it travels to the pivot's slot).  One mbarrier phase per column; buffer
    //    `par` is overwritten two columns later, after every CTA has passed the __syncthreads() that end its reads.
    {
      const double b = s_val[0];
      const int ix = s_best;
      const bool have = ix != 0x7fffffff;
      const uint32_t cbar_a = smem_u32(cbar + par);
      if (tid == 0) mbar_expect_tx(cbar + par, kColBytes);
      for (int t = tid; t < kLuCl * kLuMsg; t += kLuClThreads) {
        const int q = t / kLuMsg, x = t % kLuMsg;
        double v;
        if (x == 0) v = b;
        else if (x == 1) v = (double)ix;
        else v = (have && x - 2 < nb) ? A[(ix - r0) * kLuPad + (x - 2)] : 0.0;
        st_async_f64(mapa_u32(msg_a + (uint32_t)((((size_t)par * kLuCl + rank) * kLuMsg + x) * 8), (uint32_t)q), v,
                     mapa_u32(cbar_a, (uint32_t)q));
      }
      const int qc = (col - j0) / R;
      if (rank == qc) {
        for (int t = tid; t < kLuCl * kLuNb; t += kLuClThreads) {
          const int q = t / kLuNb, x = t % kLuNb;
          st_async_f64(mapa_u32(rowc_a + (uint32_t)(((size_t)par * kLuNb + x) * 8), (uint32_t)q),
                       x < nb ? A[(col - r0) * kLuPad + x] : 0.0, mapa_u32(cbar_a, (uint32_t)q));
        }
      }
    }
    mbar_wait(cbar + par, (uint32_t)((cc >> 1) & 1));
    // 3. everybody picks the same winner
    const double* mp = msg + (size_t)par * kLuCl * kLuMsg;
    int qw = 0;
    double pb = mp[0];
    int pr = (int)mp[1];
#pragma unroll
    for (int q = 1; q < kLuCl; ++q) {
      const double v = mp[q * kLuMsg];
      const int ix = (int)mp[q * kLuMsg + 1];
      if (v > pb || (v == pb && ix < pr)) { pb = v; pr = ix; qw = q; }
    }
    const double* prow = mp + qw * kLuMsg + 2;      // pivot row (old contents of row pr)
    const double* crow = rowc + (size_t)par * kLuNb; // old contents of row col
    const int qp = (pr - j0) / R, qc = (col - j0) / R;
    if (rank == 0 && tid == 0) {
      ipiv[col] = pr;
      if (!(pb > 0.0)) st.status = -4;  // CTAUX_ESINGULAR
      if (detsign) {
        int sg = detsign[w * 2 + sp];
        if (pr != col) sg = -sg;
        if (prow[cc] < 0.0) sg = -sg;
        detsign[w * 2 + sp] = sg;
      }
    }
    if (pr != col) {
      if (rank == qp && tid < nb) A[(pr - r0) * kLuPad + tid] = crow[tid];
      if (rank == qc && tid >= 64 && tid < 64 + nb) A[(col - r0) * kLuPad + tid - 64] = prow[tid - 64];
    }
    __syncthreads();
    // 4. elimination of the local rows below `col`
    const double piv = prow[cc];
    if (piv != 0.0) {
      for (int i = tid; i < nloc; i += kLuClThreads) {
        if (r0 + i > col) {
          double* Ai = A + i * kLuPad;
          const double l = Ai[cc] / piv;
          Ai[cc] = l;
          for (int x = cc + 1; x < nb; ++x) Ai[x] -= l * prow[x];
        }
      }
    }
    __syncthreads();
  }
  cluster.sync();   // nobody leaves while a peer may still write into its shared memory
  for (int idx = tid; idx < nloc * nb; idx += kLuClThreads) {
    const int i = idx % nloc, cc = idx / nloc;
    F[(size_t)(j0 + cc) * ld + r0 + i] = A[i * kLuPad + cc];
  }
}

// ---- rebuild_mode 1: Newton-Schulz refresh  N <- N (2 - A N) = 2 N - N (A N)
// A_sigma is built (k_build_A) into the spare N buffer; T = A N goes to Tbuf; the new N overwrites A.
struct TDescNS {
  DevCtx c;
  int stage;
  __device__ bool operator()(int prob, TmaGemmDesc& d) const {
    const int w = prob >> 1, sp = prob & 1;
    const WalkerState& st = c.ws[w];
    const int k = st.k;
    if (k == 0) return false;
    const int cur = st.n_cur, oth = st.n_cur ^ 1;
    double* T = c.Tbuf + ((size_t)w * 2 + sp) * (size_t)c.ld * c.ld;
    d.M = k; d.N = k; d.K = k;
    d.a_m0 = 0; d.a_k0 = 0; d.b_k0 = 0; d.b_n0 = 0;
    d.ldc = c.ld; d.ldc0 = c.ld; d.rowmap = nullptr; d.colmap = nullptr;
    if (stage == 0) {
      d.tmA = c.tm(w, sp, oth ? TM_N1_M : TM_N0_M); d.tmB = c.tm(w, sp, cur ? TM_N1_K : TM_N0_K);
      d.C = T; d.C0 = nullptr; d.alpha = 1.0; d.beta = 0.0;
    } else {
      d.tmA = c.tm(w, sp, cur ? TM_N1_M : TM_N0_M); d.tmB = c.tm(w, sp, TM_T_K);
      d.C = c.N(w, sp, oth); d.C0 = c.N(w, sp, cur); d.alpha = -1.0; d.beta = 2.0;
    }
    return true;
  }
};

__global__ void k_ns_resid(DevCtx c) {   // resid[prob] = max |T - 1|
  const int w = blockIdx.y >> 1, sp = blockIdx.y & 1;
  const int k = c.ws[w].k;
  const double* T = c.Tbuf + ((size_t)w * 2 + sp) * (size_t)c.ld * c.ld;
  double mx = 0.0;
  const size_t total = (size_t)k * k;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(idx % k), j = (int)(idx / k);
    const double v = fabs(T[(size_t)j * c.ld + i] - (i == j ? 1.0 : 0.0));
    mx = v > mx ? v : mx;   // NaN never wins here; it is caught below
    if (!(v == v)) mx = 1e300;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0) atomicMax(c.resid + blockIdx.y, (unsigned long long)__double_as_longlong(mx));
}

__global__ void k_ns_flip(DevCtx c) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= c.B) return;
  WalkerState& st = c.ws[w];
  if (st.k > 0) st.n_cur ^= 1;
  st.n_src = st.n_cur;
  st.rebuilds += 1;
  st.flops_rebuild += 2.0 * 4.0 * (double)st.k * st.k * st.k;   // two k^3 GEMMs per spin
}

}  // namespace ctaux

namespace ctaux {

// ===================================================================================================================
// Two-level blocking of the rebuild.  A one-level right-looking LU updates the whole trailing matrix with rank
// kLuNb = 32 after every panel: arithmetic intensity 4 flop/B, the HBM side of the FP64 ridge (5.4), and the
// forward substitution over X = L^-1 P runs over the structural zeros of the identity.  Instead:
//   * panels of 32 columns are factorised as before (partial pivoting over the full height), but their rank-32 updates
//     touch only the columns of the current OUTER block of kLuOuter = 128 columns;
//   * once per outer block: the block's 128 interchanges are applied to the rest, the 128 x 128 unit-lower block L11 is
//     inverted explicitly (|L_ij| <= 1 under partial pivoting), U12 = L11^-1 F12 and the trailing update
//     F22 -= L21 U12 run as rank-128 GEMMs on the TMA tiles (intensity 16 flop/B);
//   * X' = L^-1 is built IN POSITION SPACE instead of X = L^-1 P: it starts as the identity, receives only the
//     interchanges of rows that are not yet pivots (columns left of the block), and stays lower triangular, so the
//     forward GEMMs cover columns [0, J1) only -- k^3/3 instead of k^3 flops;
//   * backward: per outer block U11^-1 (explicit 128 x 128 inverse) and a rank-128 update of the rows above;
//   * N = N' P: one column scatter at the end (into the buffer that held F) and the buffers swap roles.
// Flops: 2/3 + 1/3 + 1 = 2 k^3, the algorithmic count.
constexpr int kLuOuter = 128;

// interchanges of the pivots [p0, min(p1, k)) applied, in order, to the F columns [fa, fb) U [fc, fd) and the X columns
// [0, xc); one thread per column
__global__ void __launch_bounds__(128) k_lu_swap_range(DevCtx c, int p0, int p1, int fa, int fb, int fc, int fd, int xc) {
  const int w = blockIdx.y >> 1, sp = blockIdx.y & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  if (p0 >= k) return;
  if (p1 > k) p1 = k;
  if (fb > k) fb = k;
  if (fd > k) fd = k;
  if (xc > k) xc = k;
  const int* ipiv = c.perm + ((size_t)w * 2 + sp) * c.ld;
  double* F = c.N(w, sp, st.n_cur ^ 1);
  double* X = c.N(w, sp, st.n_cur);
  __shared__ int s_piv[kLuOuter];
  const int np = p1 - p0;
  if (threadIdx.x < np) s_piv[threadIdx.x] = ipiv[p0 + threadIdx.x];
  __syncthreads();
  const int n1 = fb > fa ? fb - fa : 0, n2 = fd > fc ? fd - fc : 0, n3 = xc > 0 ? xc : 0;
  for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < n1 + n2 + n3; t += gridDim.x * blockDim.x) {
    double* col = t < n1 ? F + (size_t)(fa + t) * c.ld : (t < n1 + n2 ? F + (size_t)(fc + t - n1) * c.ld : X + (size_t)(t - n1 - n2) * c.ld);
    for (int q = 0; q < np; ++q) {
      const int p = s_piv[q];
      if (p != p0 + q) {
        const double a = col[p0 + q], b = col[p];
        col[p0 + q] = b;
        col[p] = a;
      }
    }
  }
}

// rows j0..j1 of the F columns [c0, min(c1, k))  <-  L11^-1 (unit lower, the 32-wide diagonal block at j0)
__global__ void __launch_bounds__(128) k_lu_trsm_range(DevCtx c, int j0, int c0, int c1) {
  constexpr int NB = kLuNb;
  const int w = blockIdx.y >> 1, sp = blockIdx.y & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  if (j0 >= k) return;
  const int j1 = (j0 + NB < k) ? j0 + NB : k;
  if (c1 > k) c1 = k;
  const int nb = j1 - j0, ld = c.ld;
  double* F = c.N(w, sp, st.n_cur ^ 1);
  __shared__ double T[NB][NB + 1];
  for (int idx = threadIdx.x; idx < nb * nb; idx += blockDim.x) {
    const int i = idx % nb, j = idx / nb;
    T[i][j] = F[(size_t)(j0 + j) * ld + j0 + i];
  }
  __syncthreads();
  for (int t = c0 + blockIdx.x * blockDim.x + threadIdx.x; t < c1; t += gridDim.x * blockDim.x) {
    double* col = F + (size_t)t * ld + j0;
    double x[NB];
#pragma unroll
    for (int i = 0; i < NB; ++i) x[i] = (i < nb) ? col[i] : 0.0;
#pragma unroll
    for (int i = 0; i < NB; ++i) {
      if (i < nb) {
        double s = x[i];
#pragma unroll
        for (int l = 0; l < NB; ++l)
          if (l < i) s -= T[i][l] * x[l];
        x[i] = s;
      }
    }
#pragma unroll
    for (int i = 0; i < NB; ++i)
      if (i < nb) col[i] = x[i];
  }
}

// explicit inverse of the diagonal block of F at J0 (size nbk = min(128, k - J0)) into Linv [128 x 128], column-major,
// leading dimension 128:  upper == 0: unit-lower L11;  upper == 1: upper-triangular U11 (with its diagonal).
// Blocked in shared memory (the column-at-a-time version spent 128 dependent global round trips per column: 107 us):
// U11 is handled as the lower-triangular U11^T and written back transposed, so one code path inverts a lower
// triangle T of 4 x 4 blocks of 32:
//   1. W_bb = T_bb^-1: one warp per diagonal block, lane j carries column j of the inverse in registers;
//   2. block sub-diagonals d = 1, 2, 3:  W_ij = -W_ii (sum_{l=j}^{i-1} T_il W_lj)   (two-sided products of 32^3).
constexpr int kTriB = 32, kTriNb = kLuOuter / kTriB;             // 4 x 4 blocks
constexpr int kTriLdT = kLuOuter + 1, kTriLdW = kTriB + 1;
constexpr int kTriSmemDoubles = kLuOuter * kTriLdT + (kTriNb * (kTriNb + 1) / 2 + 1) * kTriB * kTriLdW;
__device__ __forceinline__ int tri_blk(int i, int j) { return i * (i + 1) / 2 + j; }   // i >= j

__global__ void __launch_bounds__(512) k_lu_tri_inv(DevCtx c, double* linv_all, int J0, int upper) {
  extern __shared__ double s_T[];                 // T [128][129] (row i, column j at i*129 + j)
  double* s_W = s_T + kLuOuter * kTriLdT;        // 10 lower blocks of W [32][33] + one scratch block
  double* s_S = s_W + (kTriNb * (kTriNb + 1) / 2) * kTriB * kTriLdW;
  const int prob = blockIdx.x, w = prob >> 1, sp = prob & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  if (J0 >= k) return;
  const int nbk = (k - J0 < kLuOuter) ? k - J0 : kLuOuter;
  const double* F = c.N(w, sp, st.n_cur ^ 1);
  double* out = linv_all + (size_t)prob * kLuOuter * kLuOuter;
  const int tid = threadIdx.x;
  // load the lower triangle (of L11, or of U11^T); the padding is the identity
  for (int idx = tid; idx < kLuOuter * kLuOuter; idx += 512) {
    const int a = idx % kLuOuter, b = idx / kLuOuter;             // element (a, b) of the stored block, a fastest
    double v = (a < nbk && b < nbk) ? F[(size_t)(J0 + b) * c.ld + J0 + a] : (a == b ? 1.0 : 0.0);
    const int i = upper ? b : a, j = upper ? a : b;               // T = block (lower) or block^T (upper)
    if (i < j) v = 0.0;
    else if (i == j && !upper) v = 1.0;                           // unit diagonal (the storage holds U's there)
    s_T[i * kTriLdT + j] = v;
  }
  __syncthreads();
  // 1. diagonal blocks
  if (tid < kTriNb * 32) {
    const int b = tid >> 5, j = tid & 31;
    const double* Tb = s_T + (b * kTriB) * kTriLdT + b * kTriB;
    double x[kTriB];
#pragma unroll
    for (int i = 0; i < kTriB; ++i) {
      double s0 = (i == j) ? 1.0 : 0.0, s1 = 0.0;
#pragma unroll
      for (int l = 0; l < i; ++l) {
        if (l & 1) s1 -= Tb[i * kTriLdT + l] * x[l];
        else s0 -= Tb[i * kTriLdT + l] * x[l];
      }
      x[i] = (s0 + s1) / Tb[i * kTriLdT + i];
    }
    double* Wb = s_W + tri_blk(b, b) * kTriB * kTriLdW;
#pragma unroll
    for (int i = 0; i < kTriB; ++i) Wb[i * kTriLdW + j] = x[i];
  }
  __syncthreads();
  // 2. off-diagonal blocks, sub-diagonal by sub-diagonal; thread -> (row, two columns) of a 32 x 32 block
  const int row = tid & 31, c0 = (tid >> 5) * 2;
  for (int dgl = 1; dgl < kTriNb; ++dgl) {
    for (int i = dgl; i < kTriNb; ++i) {
      const int j = i - dgl;
      double a0 = 0.0, a1 = 0.0;
      for (int l = j; l < i; ++l) {
        const double* Til = s_T + (i * kTriB + row) * kTriLdT + l * kTriB;
        const double* Wlj = s_W + tri_blk(l, j) * kTriB * kTriLdW;
#pragma unroll 8
        for (int q = 0; q < kTriB; ++q) {
          const double t = Til[q];
          a0 += t * Wlj[q * kTriLdW + c0];
          a1 += t * Wlj[q * kTriLdW + c0 + 1];
        }
      }
      s_S[row * kTriLdW + c0] = a0;
      s_S[row * kTriLdW + c0 + 1] = a1;
      __syncthreads();
      const double* Wii = s_W + tri_blk(i, i) * kTriB * kTriLdW;
      double b0 = 0.0, b1 = 0.0;
#pragma unroll 8
      for (int q = 0; q < kTriB; ++q) {
        const double t = Wii[row * kTriLdW + q];
        b0 += t * s_S[q * kTriLdW + c0];
        b1 += t * s_S[q * kTriLdW + c0 + 1];
      }
      double* Wij = s_W + tri_blk(i, j) * kTriB * kTriLdW;
      Wij[row * kTriLdW + c0] = -b0;
      Wij[row * kTriLdW + c0 + 1] = -b1;
      __syncthreads();
    }
  }
  // write back: W (lower) or W^T (upper); zero outside the live block
  for (int idx = tid; idx < kLuOuter * kLuOuter; idx += 512) {
    const int a = idx % kLuOuter, b = idx / kLuOuter;             // out(a, b), a fastest
    const int i = upper ? b : a, j = upper ? a : b;
    double v = 0.0;
    if (i >= j && a < nbk && b < nbk) v = s_W[tri_blk(i >> 5, j >> 5) * kTriB * kTriLdW + (i & 31) * kTriLdW + (j & 31)];
    out[idx] = v;
  }
}

// rows J0..J1 back from the scratch `tmp` [128][ld] (row i, column cidx at tmp[i + cidx*128]):
//   mode 0 (forward):  F[J0:J1, J1:k) = tmp,  X[J0:J1, 0:J0) = tmp,  X[J0:J1, J0:J1) = Linv
//   mode 1 (backward): X[J0:J1, 0:k) = tmp
__global__ void k_lu_copyback(DevCtx c, const double* tmp_all, const double* linv_all, int J0, int mode) {
  const int prob = blockIdx.y, w = prob >> 1, sp = prob & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  if (J0 >= k) return;
  const int nbk = (k - J0 < kLuOuter) ? k - J0 : kLuOuter, J1 = J0 + nbk;
  double* F = c.N(w, sp, st.n_cur ^ 1);
  double* X = c.N(w, sp, st.n_cur);
  const double* tmp = tmp_all + (size_t)prob * kLuOuter * c.ld;
  const double* linv = linv_all + (size_t)prob * kLuOuter * kLuOuter;
  const size_t total = (size_t)nbk * k;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(idx % nbk), cidx = (int)(idx / nbk);
    if (mode == 1) X[(size_t)cidx * c.ld + J0 + i] = tmp[(size_t)cidx * kLuOuter + i];
    else if (cidx >= J1) F[(size_t)cidx * c.ld + J0 + i] = tmp[(size_t)cidx * kLuOuter + i];
    else if (cidx < J0) X[(size_t)cidx * c.ld + J0 + i] = tmp[(size_t)cidx * kLuOuter + i];
    else X[(size_t)cidx * c.ld + J0 + i] = linv[(size_t)(cidx - J0) * kLuOuter + i];
  }
}

// row permutation of P A = L U as an index array: pos[i] = original row that sits in position i
__global__ void k_lu_perm(DevCtx c, int32_t* pos_all) {
  const int prob = blockIdx.x * blockDim.x + threadIdx.x;
  if (prob >= 2 * c.B) return;
  const int w = prob >> 1, sp = prob & 1;
  const int k = c.ws[w].k;
  const int* ipiv = c.perm + ((size_t)w * 2 + sp) * c.ld;
  int32_t* pos = pos_all + (size_t)prob * c.ld;
  for (int i = 0; i < k; ++i) pos[i] = i;
  for (int j = 0; j < k; ++j) {
    const int p = ipiv[j];
    if (p != j) { const int a = pos[j]; pos[j] = pos[p]; pos[p] = a; }
  }
}
// N = N' P:  N[:, pos[i]] = N'[:, i], written into the buffer that held the LU factors
__global__ void k_lu_scatter_cols(DevCtx c, const int32_t* pos_all) {
  const int prob = blockIdx.y, w = prob >> 1, sp = prob & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  const double* X = c.N(w, sp, st.n_cur);
  double* O = c.N(w, sp, st.n_cur ^ 1);
  const int32_t* pos = pos_all + (size_t)prob * c.ld;
  const size_t total = (size_t)k * k;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(idx % k), j = (int)(idx / k);
    O[(size_t)pos[j] * c.ld + i] = X[(size_t)j * c.ld + i];
  }
}
__global__ void k_lu_flip(DevCtx c) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= c.B) return;
  WalkerState& st = c.ws[w];
  if (st.k > 0) st.n_cur ^= 1;
  st.n_src = st.n_cur;
}

// GEMM problems of the two-level LU (alpha = -1, beta = 1 in place, or alpha = 1, beta = 0 into the row scratch).
//   0: F[j1:, j1:J1) -= F[j1:, j0:j1) F[j0:j1, j1:J1)                (inner, rank <= 32, inside the outer block)
//   1: tmp[:, J1:k)   = Linv F[J0:J1, J1:k)         2: tmp[:, 0:J0) = Linv X[J0:J1, 0:J0)
//   3: F[J1:, J1:)   -= F[J1:, J0:J1) F[J0:J1, J1:)  4: X[J1:, 0:J1) -= F[J1:, J0:J1) X[J0:J1, 0:J1)
//   5: tmp[:, 0:k)    = Uinv X[J0:J1, 0:k)           6: X[0:J0, 0:k) -= F[0:J0, J0:J1) X[J0:J1, 0:k)
// A launch covers `which_a` for problems [0, 2B) and `which_b` (if >= 0) for problems [2B, 4B).
struct TDescLU2 {
  DevCtx c;
  int J0, j0, which_a, which_b;
  double* tmp_all;
  __device__ bool operator()(int prob, TmaGemmDesc& d) const {
    const int P = 2 * c.B;
    const int which = prob < P ? which_a : which_b;
    if (prob >= P) prob -= P;
    if (which < 0) return false;
    const int w = prob >> 1, sp = prob & 1;
    const WalkerState& st = c.ws[w];
    const int k = st.k;
    if (J0 >= k) return false;
    const int J1 = (J0 + kLuOuter < k) ? J0 + kLuOuter : k;
    const size_t ld = c.ld;
    const int fb = st.n_cur ^ 1, xb = st.n_cur;
    double* F = c.N(w, sp, fb);
    double* X = c.N(w, sp, xb);
    double* tmp = tmp_all + (size_t)prob * kLuOuter * c.ld;
    const CUtensorMap *FM = c.tm(w, sp, fb ? TM_N1_M : TM_N0_M), *FK = c.tm(w, sp, fb ? TM_N1_K : TM_N0_K);
    const CUtensorMap* XK = c.tm(w, sp, xb ? TM_N1_K : TM_N0_K);
    d.rowmap = nullptr; d.colmap = nullptr;
    d.alpha = -1.0; d.beta = 1.0; d.ldc = c.ld; d.ldc0 = c.ld;
    if (which == 0) {
      if (j0 >= k) return false;
      const int j1 = (j0 + kLuNb < k) ? j0 + kLuNb : k;
      d.M = k - j1; d.N = J1 - j1; d.K = j1 - j0;
      d.tmA = FM; d.a_m0 = j1; d.a_k0 = j0; d.tmB = FK; d.b_k0 = j0; d.b_n0 = j1;
      d.C = F + j1 + (size_t)j1 * ld;
    } else if (which == 1 || which == 2 || which == 5) {
      d.M = J1 - J0; d.K = J1 - J0;
      d.tmA = c.tm(w, sp, TM_LINV_M); d.a_m0 = 0; d.a_k0 = 0;
      d.b_k0 = J0;
      if (which == 1) { d.N = k - J1; d.tmB = FK; d.b_n0 = J1; d.C = tmp + (size_t)J1 * kLuOuter; }
      else if (which == 2) { d.N = J0; d.tmB = XK; d.b_n0 = 0; d.C = tmp; }
      else { d.N = k; d.tmB = XK; d.b_n0 = 0; d.C = tmp; }
      d.alpha = 1.0; d.beta = 0.0; d.ldc = kLuOuter; d.ldc0 = 0;
      d.C0 = nullptr;
      return d.M > 0 && d.N > 0;
    } else if (which == 3) {
      d.M = k - J1; d.N = k - J1; d.K = J1 - J0;
      d.tmA = FM; d.a_m0 = J1; d.a_k0 = J0; d.tmB = FK; d.b_k0 = J0; d.b_n0 = J1;
      d.C = F + J1 + (size_t)J1 * ld;
    } else if (which == 4) {
      d.M = k - J1; d.N = J1; d.K = J1 - J0;
      d.tmA = FM; d.a_m0 = J1; d.a_k0 = J0; d.tmB = XK; d.b_k0 = J0; d.b_n0 = 0;
      d.C = X + J1;
    } else {
      d.M = J0; d.N = k; d.K = J1 - J0;
      d.tmA = FM; d.a_m0 = 0; d.a_k0 = J0; d.tmB = XK; d.b_k0 = J0; d.b_n0 = 0;
      d.C = X;
    }
    d.C0 = d.C;
    return d.M > 0 && d.N > 0;
  }
};

}  // namespace ctaux
