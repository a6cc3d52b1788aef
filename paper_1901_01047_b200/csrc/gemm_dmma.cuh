// Grouped FP64 GEMM on the sm_100a FP64 tensor pipe (mma.sync m8n8k4 -> SASS DMMA.8x8x4).
//
// Serves S2 (candidate rows / columns), S4 (U*S^-1 and the rank-r flush with its compaction
// gather) and S5 (trailing updates of the blocked LU).  PAPER.md:226 ("rank-k_s operation"),
// PAPER.md:373 ("large matrix-matrix multiplications").
//
// All operands are column-major.  One launch covers a GROUP of independent problems
// (walker x spin); each problem's sizes and pointers come from a device-side descriptor
// that a functor builds from the walker state, so no host round trip is needed when the
// expansion order changes.
//
//   C[i,j] = beta * C0[rowmap[i], colmap[j]] + alpha * sum_k A[i,k] * B[k,j]
//
// Tiling: CTA tile BM x BN x 16, 256 threads = 8 warps, cp.async (16-byte, zero-filled
// tails) multi-stage pipeline into shared memory; each warp owns a (BM/WM) x (BN/WN) tile of
// 8x8 DMMA fragments held in registers.
//   A_s[k][m]  (m contiguous, row stride BM+4): fragment reads hit 16 distinct 8-byte banks
//   B_s[n][k]  (k contiguous, row stride 20)  : same
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ctaux {

struct GemmDesc {
  int M, N, K;
  const double* A; int lda;      // M x K
  const double* B; int ldb;      // K x N
  double* C; int ldc;            // M x N
  const double* C0; int ldc0;    // source of the beta term (may alias C when no maps are given)
  const int* rowmap;             // nullptr = identity
  const int* colmap;
  double alpha, beta;
};

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

template <int BM, int BN, int WM, int WN, int STAGES>
struct GemmCfg {
  static constexpr int BK = 16;
  static constexpr int THREADS = WM * WN * 32;
  static constexpr int LDA_S = BM + 4;   // doubles
  static constexpr int LDB_S = BK + 4;
  static constexpr int A_STAGE = BK * LDA_S;
  static constexpr int B_STAGE = BN * LDB_S;
  static constexpr int SMEM_BYTES = STAGES * (A_STAGE + B_STAGE) * 8;
  static constexpr int TM = BM / WM / 8;  // 8x8 fragments per warp along M
  static constexpr int TN = BN / WN / 8;
};

// One CTA computes one BM x BN tile of one problem.
template <int BM, int BN, int WM, int WN, int STAGES, bool PRE = false>
__device__ __forceinline__ void gemm_tile(const GemmDesc& d, int tile_m, int tile_n, double* smem,
                                          const int* pre_srow = nullptr, const int* pre_scol = nullptr) {
  using Cfg = GemmCfg<BM, BN, WM, WN, STAGES>;
  constexpr int BK = Cfg::BK, LDA_S = Cfg::LDA_S, LDB_S = Cfg::LDB_S;
  constexpr int TM = Cfg::TM, TN = Cfg::TN, THREADS = Cfg::THREADS;
  double* As = smem;
  double* Bs = smem + STAGES * Cfg::A_STAGE;

  const int tid = threadIdx.x;
  const int warp = tid >> 5, lane = tid & 31;
  const int wm = warp % WM, wn = warp / WM;
  const int g = lane >> 2, q = lane & 3;
  const int m0 = tile_m * BM, n0 = tile_n * BN;
  const int M = d.M, N = d.N, K = d.K;

  // index maps of this thread's fragment rows / columns (C0 gather = compaction of the flush)
  int crow[TM], srow[TM], ccol[TN][2], scol[TN][2];
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    crow[i] = m0 + wm * (TM * 8) + i * 8 + g;
    if (PRE) srow[i] = pre_srow[i];
    else srow[i] = (d.rowmap && crow[i] < M) ? d.rowmap[crow[i]] : crow[i];
  }
#pragma unroll
  for (int j = 0; j < TN; ++j)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      ccol[j][h] = n0 + wn * (TN * 8) + j * 8 + 2 * q + h;
      if (PRE) scol[j][h] = pre_scol[j * 2 + h];
      else scol[j][h] = (d.colmap && ccol[j][h] < N) ? d.colmap[ccol[j][h]] : ccol[j][h];
    }
  const int nk = (K + BK - 1) / BK;

  auto load_stage = [&](int kt, int st) {
    const int k0 = kt * BK;
    // A tile: BK columns (k) x BM rows (m), 16-byte chunks along m
    constexpr int A_CHUNKS = BK * BM / 2;
#pragma unroll
    for (int c = tid; c < A_CHUNKS; c += THREADS) {
      const int kk = c / (BM / 2), mm = (c % (BM / 2)) * 2;
      const int gk = k0 + kk, gm = m0 + mm;
      int bytes = 0;
      if (gk < K) bytes = (gm + 1 < M) ? 16 : ((gm < M) ? 8 : 0);
      const double* src = bytes ? (d.A + (size_t)gk * d.lda + gm) : d.A;
      cp_async16(As + st * Cfg::A_STAGE + kk * LDA_S + mm, src, bytes);
    }
    // B tile: BN columns (n) x BK rows (k), 16-byte chunks along k
    constexpr int B_CHUNKS = BN * BK / 2;
#pragma unroll
    for (int c = tid; c < B_CHUNKS; c += THREADS) {
      const int nn = c / (BK / 2), kk = (c % (BK / 2)) * 2;
      const int gk = k0 + kk, gn = n0 + nn;
      int bytes = 0;
      if (gn < N) bytes = (gk + 1 < K) ? 16 : ((gk < K) ? 8 : 0);
      const double* src = bytes ? (d.B + (size_t)gn * d.ldb + gk) : d.B;
      cp_async16(Bs + st * Cfg::B_STAGE + nn * LDB_S + kk, src, bytes);
    }
  };

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < nk) load_stage(s, s);
    cp_async_commit();
  }

  // Accumulators start from C0[gather] (scaled by beta/alpha when that is not 1): the loads are in
  // flight while the pipeline fills and the epilogue is a pure store.  The common in-place update
  // C = C0 - A*B (alpha = -1, beta = 1: flush, LU trailing updates) flips the sign bit of the A
  // fragments instead, so the C0 values go straight into the accumulator registers.
  const bool negA = (d.alpha == -1.0 && d.beta == 1.0);
  const double alpha_eff = negA ? 1.0 : d.alpha;
  double acc[TM][TN][2];
  if (d.beta != 0.0) {
    const double bscale = d.beta / alpha_eff;
#pragma unroll
    for (int j = 0; j < TN; ++j)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const double* c0col = d.C0 + (size_t)scol[j][h] * d.ldc0;
        const bool cok = ccol[j][h] < N;
#pragma unroll
        for (int i = 0; i < TM; ++i) acc[i][j][h] = (cok && crow[i] < M) ? c0col[srow[i]] : 0.0;
      }
    if (bscale != 1.0) {
#pragma unroll
      for (int j = 0; j < TN; ++j)
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
          for (int i = 0; i < TM; ++i) acc[i][j][h] *= bscale;
    }
  } else {
#pragma unroll
    for (int j = 0; j < TN; ++j)
#pragma unroll
      for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int i = 0; i < TM; ++i) acc[i][j][h] = 0.0;
  }
  const int sign_flip = negA ? (int)0x80000000 : 0;

  for (int kt = 0; kt < nk; ++kt) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    {
      const int nxt = kt + STAGES - 1;
      if (nxt < nk) load_stage(nxt, nxt % STAGES);
      cp_async_commit();
    }
    const double* a_s = As + (kt % STAGES) * Cfg::A_STAGE + wm * (TM * 8) + g;
    const double* b_s = Bs + (kt % STAGES) * Cfg::B_STAGE + (wn * (TN * 8) + g) * LDB_S;
#pragma unroll
    for (int k4 = 0; k4 < BK; k4 += 4) {
      double af[TM], bf[TN];
#pragma unroll
      for (int i = 0; i < TM; ++i) {
        const double a = a_s[(k4 + q) * LDA_S + i * 8];
        af[i] = __hiloint2double(__double2hiint(a) ^ sign_flip, __double2loint(a));
      }
#pragma unroll
      for (int j = 0; j < TN; ++j) bf[j] = b_s[j * 8 * LDB_S + k4 + q];
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    }
  }
  cp_async_wait<0>();

  // epilogue: thread holds C[row = g][cols 2q, 2q+1] of every 8x8 fragment
#pragma unroll
  for (int j = 0; j < TN; ++j)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      if (ccol[j][h] >= N) continue;
      double* ccolp = d.C + (size_t)ccol[j][h] * d.ldc;
#pragma unroll
      for (int i = 0; i < TM; ++i)
        if (crow[i] < M) ccolp[crow[i]] = (alpha_eff == 1.0) ? acc[i][j][h] : alpha_eff * acc[i][j][h];
    }
}

// L2 prefetch of the beta*C0[gather] tile that will run in this SM slot a wave later.  The flush is an
// in-place-style rank-r update (K = r <= 64): each tile reads 64 KB of N from HBM for ~1 MFLOP, so the
// C0 gather sits on the critical path of every CTA; pulling the lines into L2 one wave ahead turns
// those loads into L2 hits (rank-k_s update; 16 n^2 bytes per 2 n^2 r flops).
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p)); }

template <int BM, int BN, int THREADS>
__device__ __forceinline__ void prefetch_c0_tile(const GemmDesc& d, int tile_m, int tile_n) {
  const int m0 = tile_m * BM, n0 = tile_n * BN;
  constexpr int RG = BM / 16;   // one 128-byte line = 16 doubles
  for (int idx = threadIdx.x; idx < BN * RG; idx += THREADS) {
    const int col = n0 + idx / RG, row = m0 + (idx % RG) * 16;
    if (col >= d.N || row >= d.M) continue;
    const int sr = d.rowmap ? __ldg(d.rowmap + row) : row;
    const int sc = d.colmap ? __ldg(d.colmap + col) : col;
    prefetch_l2(d.C0 + (size_t)sc * d.ldc0 + sr);
  }
}

// Grouped launch: blockIdx.y = problem, blockIdx.x = tile (tiles beyond the problem's own
// count exit).  DescFn(problem) -> GemmDesc, evaluated on the device.
template <int BM, int BN, int WM, int WN, int STAGES, int MINB, class DescFn>
__global__ void __launch_bounds__(WM * WN * 32, MINB) gemm_grouped_kernel(DescFn fn, int pf_dist) {
  extern __shared__ __align__(16) double smem_gemm[];
  GemmDesc d;
  if (!fn(blockIdx.y, d)) return;
  if (d.M <= 0 || d.N <= 0) return;
  const int tm = (d.M + BM - 1) / BM, tn = (d.N + BN - 1) / BN;
  // persistent over the tiles of this problem: grid.x CTAs stride over tm*tn tiles
  for (int t = blockIdx.x; t < tm * tn; t += gridDim.x) {
    if (d.beta != 0.0 && pf_dist > 0) {
      int t2 = t + pf_dist;
      if (t2 < tm * tn) {
        prefetch_c0_tile<BM, BN, WM * WN * 32>(d, t2 % tm, t2 / tm);
      } else if (blockIdx.y + 1 < gridDim.y) {
        GemmDesc d2;
        t2 -= tm * tn;
        if (fn(blockIdx.y + 1, d2) && d2.M > 0 && d2.N > 0 && d2.beta != 0.0) {
          const int tm2 = (d2.M + BM - 1) / BM, tn2 = (d2.N + BN - 1) / BN;
          if (t2 < tm2 * tn2) prefetch_c0_tile<BM, BN, WM * WN * 32>(d2, t2 % tm2, t2 / tm2);
        }
      }
    }
    gemm_tile<BM, BN, WM, WN, STAGES>(d, t % tm, t / tm, smem_gemm);
    __syncthreads();
  }
}

// Flush form of the grouped kernel: the tile -> (tile_m, tile_n) mapping uses a host-side tile count `tmax`
// instead of the problem's own size, so every CTA can issue the loads of its compaction-map entries
// (map of problem p at maps + (p >> 1) * map_stride, rows and columns alike) BEFORE the device-side descriptor
// has arrived: the dependent chain  descriptor -> maps -> C0  loses one L2 round trip per CTA.
// Tiles beyond the live size exit.  The host's tile count comes from a hint of the live order that can be stale
// (the order grows by up to `delay` per block step between two polls): when the problem has more tiles than
// tmax x tmax, the CTAs of the launch stride over the uncovered ones afterwards, so a stale hint costs balance,
// never correctness.  Speculative map reads are clamped to the walker's own map (map_stride entries).
template <int BM, int BN, int WM, int WN, int STAGES, int MINB, class DescFn>
__global__ void __launch_bounds__(WM * WN * 32, MINB)
    gemm_flush_kernel(DescFn fn, const int* maps, int map_stride, int tmax) {
  extern __shared__ __align__(16) double smem_gemm[];
  using Cfg = GemmCfg<BM, BN, WM, WN, STAGES>;
  constexpr int TM = Cfg::TM, TN = Cfg::TN;
  const int tile_m = blockIdx.x % tmax, tile_n = blockIdx.x / tmax;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int wm = warp % WM, wn = warp / WM, g = lane >> 2, q = lane & 3;
  const int* map = maps + (size_t)(blockIdx.y >> 1) * map_stride;
  int psrow[TM], pscol[TN * 2];
#pragma unroll
  for (int i = 0; i < TM; ++i) psrow[i] = __ldg(map + min(tile_m * BM + wm * (TM * 8) + i * 8 + g, map_stride - 1));
#pragma unroll
  for (int j = 0; j < TN; ++j)
#pragma unroll
    for (int h = 0; h < 2; ++h)
      pscol[j * 2 + h] = __ldg(map + min(tile_n * BN + wn * (TN * 8) + j * 8 + 2 * q + h, map_stride - 1));
  GemmDesc d;
  if (!fn(blockIdx.y, d)) return;
  if (tile_m * BM < d.M && tile_n * BN < d.N)
    gemm_tile<BM, BN, WM, WN, STAGES, true>(d, tile_m, tile_n, smem_gemm, psrow, pscol);
  const int tm = (d.M + BM - 1) / BM, tn = (d.N + BN - 1) / BN;
  if (tm <= tmax && tn <= tmax) return;
  // uncovered tiles: rows of tiles at or beyond tmax (all columns), then columns at or beyond tmax of the covered rows
  const int rows_x = tm > tmax ? tm - tmax : 0, cols_x = tn > tmax ? tn - tmax : 0;
  const int tm_cov = tm < tmax ? tm : tmax;
  const int extra = rows_x * tn + tm_cov * cols_x;
  for (int e = blockIdx.x; e < extra; e += gridDim.x) {
    int em, en;
    if (e < rows_x * tn) { em = tmax + e % rows_x; en = e / rows_x; }
    else { const int f = e - rows_x * tn; em = f % tm_cov; en = tmax + f / tm_cov; }
    __syncthreads();   // the shared-memory ring of the previous tile is free
    gemm_tile<BM, BN, WM, WN, STAGES>(d, em, en, smem_gemm);
  }
}

}  // namespace ctaux
