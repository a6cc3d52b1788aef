// S5: from-scratch rebuild  N_sigma = A_sigma^{-1}  by blocked right-looking LU with partial
// pivoting, batched over all B*2 matrices (each with its own order k), followed by blocked
// forward / backward substitution on the identity.  BASELINE.json: "a batched LU-based rebuild".
//
//   F = the non-current N buffer (A, overwritten by its LU factors: P A = L U)
//   X = the current N buffer     (starts as I; row swaps make it P; then L^-1 P; then U^-1 L^-1 P)
//
// Per panel [j0, j1) of kLuNb columns:
//   k_lu_panel : unblocked LU of the panel with partial pivoting (one CTA per matrix)
//   k_lu_swap  : the panel's row interchanges applied to F outside the panel and to all of X
//   k_lu_trsm  : rows j0..j1 of F (right of the panel) and of X  <-  L11^-1 * (those rows)
//   GEMM       : trailing update of F (A22 -= L21 U12) and of X (X_below -= L21 X_panel)
// Backward pass, panels from last to first:
//   k_lu_trsm (upper) : X[j0:j1, :] <- U11^-1 X[j0:j1, :]
//   GEMM              : X[0:j0, :] -= U[0:j0, j0:j1] X[j0:j1, :]
// The trailing updates run on the DMMA GEMM tiles of gemm_dmma.cuh.
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

template <int NB>   // panel width: 64 when the slabs fit shared memory (config 4), else 32
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
    //    of row `col` also sends that row (it travels to the pivot's slot).  One cluster barrier per column.
    {
      const double b = s_val[0];
      const int ix = s_best;
      const bool have = ix != 0x7fffffff;
      for (int t = tid; t < kLuCl * kLuMsg; t += kLuClThreads) {
        const int q = t / kLuMsg, x = t % kLuMsg;
        double* dst = cluster.map_shared_rank(msg, q) + ((size_t)par * kLuCl + rank) * kLuMsg;
        double v;
        if (x == 0) v = b;
        else if (x == 1) v = (double)ix;
        else v = (have && x - 2 < nb) ? A[(ix - r0) * kLuPad + (x - 2)] : 0.0;
        dst[x] = v;
      }
      const int qc = (col - j0) / R;
      if (rank == qc) {
        for (int t = tid; t < kLuCl * kLuNb; t += kLuClThreads) {
          const int q = t / kLuNb, x = t % kLuNb;
          double* dst = cluster.map_shared_rank(rowc, q) + (size_t)par * kLuNb;
          dst[x] = x < nb ? A[(col - r0) * kLuPad + x] : 0.0;
        }
      }
    }
    cluster.sync();
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

// one thread per column: apply the panel's interchanges to F (outside the panel) and to X (all columns)
template <int NB>
__global__ void k_lu_swap(DevCtx c, int j0) {
  constexpr int kLuNb = NB;
  const int w = blockIdx.y >> 1, sp = blockIdx.y & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  if (j0 >= k) return;
  const int j1 = (j0 + kLuNb < k) ? j0 + kLuNb : k;
  const int* ipiv = c.perm + ((size_t)w * 2 + sp) * c.ld;
  double* F = c.N(w, sp, st.n_cur ^ 1);
  double* X = c.N(w, sp, st.n_cur);
  __shared__ int s_piv[kLuNb];
  if (threadIdx.x < j1 - j0) s_piv[threadIdx.x] = ipiv[j0 + threadIdx.x];
  __syncthreads();
  for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < 2 * k; t += gridDim.x * blockDim.x) {
    double* col;
    if (t < k) {
      if (t >= j0 && t < j1) continue;
      col = F + (size_t)t * c.ld;
    } else {
      col = X + (size_t)(t - k) * c.ld;
    }
    for (int q = 0; q < j1 - j0; ++q) {
      const int p = s_piv[q];
      if (p != j0 + q) {
        const double a = col[j0 + q], b = col[p];
        col[j0 + q] = b;
        col[p] = a;
      }
    }
  }
}

// Triangular solves with the kLuNb x kLuNb diagonal block, one thread per right-hand-side column.
//   upper == 0: rows j0..j1 of F (columns >= j1) and of X (all columns)  <-  L11^-1 (unit lower)
//   upper == 1: rows j0..j1 of X (all columns)                           <-  U11^-1
template <int NB>
__global__ void __launch_bounds__(128) k_lu_trsm(DevCtx c, int j0, int upper) {
  constexpr int kLuNb = NB;
  const int w = blockIdx.y >> 1, sp = blockIdx.y & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  if (j0 >= k) return;
  const int j1 = (j0 + kLuNb < k) ? j0 + kLuNb : k;
  const int nb = j1 - j0, ld = c.ld;
  double* F = c.N(w, sp, st.n_cur ^ 1);
  double* X = c.N(w, sp, st.n_cur);
  __shared__ double T[kLuNb][kLuNb + 1];
  for (int idx = threadIdx.x; idx < nb * nb; idx += blockDim.x) {
    const int i = idx % nb, j = idx / nb;
    T[i][j] = F[(size_t)(j0 + j) * ld + j0 + i];
  }
  __syncthreads();
  const int ncolF = upper ? 0 : (k - j1);
  const int total = ncolF + k;
  for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < total; t += gridDim.x * blockDim.x) {
    double* col = (t < ncolF) ? (F + (size_t)(j1 + t) * ld + j0) : (X + (size_t)(t - ncolF) * ld + j0);
    double x[kLuNb];
#pragma unroll
    for (int i = 0; i < kLuNb; ++i) x[i] = (i < nb) ? col[i] : 0.0;
    if (!upper) {
#pragma unroll
      for (int i = 0; i < kLuNb; ++i) {
        if (i < nb) {
          double s = x[i];
#pragma unroll
          for (int l = 0; l < kLuNb; ++l)
            if (l < i) s -= T[i][l] * x[l];
          x[i] = s;
        }
      }
    } else {
#pragma unroll
      for (int i = kLuNb - 1; i >= 0; --i) {
        if (i < nb) {
          double s = x[i];
#pragma unroll
          for (int l = 0; l < kLuNb; ++l)
            if (l > i && l < nb) s -= T[i][l] * x[l];
          x[i] = s / T[i][i];
        }
      }
    }
#pragma unroll
    for (int i = 0; i < kLuNb; ++i)
      if (i < nb) col[i] = x[i];
  }
}

// GEMM descriptors of the trailing updates (alpha = -1, beta = 1, in place)
struct TDescLU {   // operands by tensor map + tile origin (gemm_tma.cuh); j0, j1 are multiples of the panel width 32
  DevCtx c;
  int j0, which, nb;
  __device__ bool operator()(int prob, TmaGemmDesc& d) const {
    const int w = prob >> 1, sp = prob & 1;
    const WalkerState& st = c.ws[w];
    const int k = st.k;
    if (j0 >= k) return false;
    const int j1 = (j0 + nb < k) ? j0 + nb : k;
    const size_t ld = c.ld;
    const int fb = st.n_cur ^ 1, xb = st.n_cur;     // F = the non-current buffer, X = the current one
    double* F = c.N(w, sp, fb);
    double* X = c.N(w, sp, xb);
    d.K = j1 - j0;
    d.ldc = c.ld; d.ldc0 = c.ld; d.rowmap = nullptr; d.colmap = nullptr; d.alpha = -1.0; d.beta = 1.0;
    d.tmA = c.tm(w, sp, fb ? TM_N1_M : TM_N0_M); d.a_k0 = j0;
    d.b_k0 = j0;
    if (which == 0) {
      d.M = k - j1; d.N = k - j1; d.a_m0 = j1;
      d.tmB = c.tm(w, sp, fb ? TM_N1_K : TM_N0_K); d.b_n0 = j1;
      d.C = F + j1 + (size_t)j1 * ld;
    } else if (which == 1) {
      d.M = k - j1; d.N = k; d.a_m0 = j1;
      d.tmB = c.tm(w, sp, xb ? TM_N1_K : TM_N0_K); d.b_n0 = 0;
      d.C = X + j1;
    } else {
      d.M = j0; d.N = k; d.a_m0 = 0;
      d.tmB = c.tm(w, sp, xb ? TM_N1_K : TM_N0_K); d.b_n0 = 0;
      d.C = X;
    }
    d.C0 = d.C;
    return d.M > 0 && d.N > 0;
  }
};

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
