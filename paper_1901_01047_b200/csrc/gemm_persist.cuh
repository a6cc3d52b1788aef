// Persistent grouped FP64 GEMM for the large-k configurations (configs 4-5: few big matrices).
//
// Same contract as gemm_dmma.cuh (column-major, device-side descriptors, DMMA.8x8x4 through
// mma.sync m8n8k4), different schedule:
//   * ONE CTA per SM with 16 warps (the DMMA pipe needs >= 4 warps per scheduler to stay busy:
//     measured 62 % of peak with 8 warps, see profiles/), each CTA walks a strided list of tiles
//     drawn from ALL problems of the launch (prefix sum of per-problem tile counts in shared memory);
//   * K is consumed in steps of BK through a STAGES-deep cp.async ring that runs ACROSS tiles: the
//     operands of the first steps of tile t+1 land while the DMMAs of tile t still run;
//   * the beta*C0[gather] term of tile t+1 is prefetched into registers three k-steps before tile t
//     ends, so for the rank-r flush (K = r <= 64) the HBM read of N, the DMMA work and the HBM write
//     of N overlap inside one CTA.  PAPER.md:226 (rank-k_s update), PAPER.md:373 (the GPU work is
//     these matrix-matrix products).
//   * two tile orientations in one kernel (128x64 and 64x128, warp tile 32x16 in both), chosen per
//     problem by the descriptor, so that skinny operands (m = 64 candidate rows) waste no tile.
#pragma once
#include "gemm_dmma.cuh"

namespace ctaux {

constexpr int kPThreads = 512;
constexpr int kPMaxProblems = 64;

template <int BK, int STAGES>
struct PCfg {
  static constexpr int STAGE_N = BK * (128 + 4) + 64 * (BK + 4);    // 128x64 orientation
  static constexpr int STAGE_W = BK * (64 + 4) + 128 * (BK + 4);    // 64x128 orientation
  static constexpr int STAGE_DOUBLES = STAGE_N > STAGE_W ? STAGE_N : STAGE_W;
  static constexpr int SMEM_BYTES = STAGES * STAGE_DOUBLES * 8;
};

struct PTileRef {
  int p;         // problem
  int m0, n0;
  int nk;        // k-steps
};

template <int BM, int BN, int BK>
struct POrient {
  static constexpr int WM = BM / 32, WN = BN / 16;     // 4x4 or 2x8 warps, warp tile 32x16
  static constexpr int LDA_S = BM + 4, LDB_S = BK + 4;
  static constexpr int A_STAGE = BK * LDA_S;
};

// cp.async of k-step `ks` of a tile into one stage buffer (every 16-byte chunk of the stage is
// written: data, or zeros outside the matrix)
template <int BM, int BN, int BK>
__device__ __forceinline__ void p_load_step(const GemmDesc& d, const PTileRef& t, int ks, double* stage) {
  using O = POrient<BM, BN, BK>;
  const int tid = threadIdx.x;
  const int k0 = ks * BK;
  double* As = stage;
  double* Bs = stage + O::A_STAGE;
  constexpr int A_CPR = BM / 2;                // 16-byte chunks per k row
#pragma unroll
  for (int c = tid; c < BK * A_CPR; c += kPThreads) {
    const int kk = c / A_CPR, mm = (c % A_CPR) * 2;
    const int gk = k0 + kk, gm = t.m0 + mm;
    int bytes = 0;
    if (gk < d.K) bytes = (gm + 1 < d.M) ? 16 : ((gm < d.M) ? 8 : 0);
    const double* src = bytes ? (d.A + (size_t)gk * d.lda + gm) : d.A;
    cp_async16(As + kk * O::LDA_S + mm, src, bytes);
  }
  constexpr int B_CPR = BK / 2;                // 16-byte chunks per n row
#pragma unroll
  for (int c = tid; c < BN * B_CPR; c += kPThreads) {
    const int nn = c / B_CPR, kk = (c % B_CPR) * 2;
    const int gk = k0 + kk, gn = t.n0 + nn;
    int bytes = 0;
    if (gn < d.N) bytes = (gk + 1 < d.K) ? 16 : ((gk < d.K) ? 8 : 0);
    const double* src = bytes ? (d.B + (size_t)gn * d.ldb + gk) : d.B;
    cp_async16(Bs + nn * O::LDB_S + kk, src, bytes);
  }
}

// beta-scaled C0[gather] of a tile into fragment registers (issued early, consumed a tile later)
template <int BM, int BN, int BK>
__device__ __forceinline__ void p_fetch_c0(const GemmDesc& d, const PTileRef& t, double (&v)[4][2][2]) {
  using O = POrient<BM, BN, BK>;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int wm = warp % O::WM, wn = warp / O::WM;
  const int g = lane >> 2, q = lane & 3;
  if (d.beta == 0.0) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 2; ++j) { v[i][j][0] = 0.0; v[i][j][1] = 0.0; }
    return;
  }
  int srow[4];
  bool rok[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = t.m0 + wm * 32 + i * 8 + g;
    rok[i] = r < d.M;
    srow[i] = (d.rowmap && rok[i]) ? __ldg(d.rowmap + r) : r;
  }
#pragma unroll
  for (int j = 0; j < 2; ++j)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int cc = t.n0 + wn * 16 + j * 8 + 2 * q + h;
      const bool cok = cc < d.N;
      const int sc = (d.colmap && cok) ? __ldg(d.colmap + cc) : cc;
      const double* c0col = d.C0 + (size_t)sc * d.ldc0;
#pragma unroll
      for (int i = 0; i < 4; ++i) v[i][j][h] = (cok && rok[i]) ? c0col[srow[i]] : 0.0;
    }
}

template <int BM, int BN, int BK>
__device__ __forceinline__ void p_compute_step(const double* stage, double (&acc)[4][2][2], int sign_flip) {
  using O = POrient<BM, BN, BK>;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int wm = warp % O::WM, wn = warp / O::WM;
  const int g = lane >> 2, q = lane & 3;
  const double* a_s = stage + wm * 32 + g + q * O::LDA_S;
  const double* b_s = stage + O::A_STAGE + (wn * 16 + g) * O::LDB_S + q;
#pragma unroll
  for (int k4 = 0; k4 < BK; k4 += 4) {
    double af[4], bf[2];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const double a = a_s[k4 * O::LDA_S + i * 8];
      af[i] = __hiloint2double(__double2hiint(a) ^ sign_flip, __double2loint(a));
    }
#pragma unroll
    for (int j = 0; j < 2; ++j) bf[j] = b_s[j * 8 * O::LDB_S + k4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 2; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
  }
}

template <int BM, int BN, int BK>
__device__ __forceinline__ void p_store(const GemmDesc& d, const PTileRef& t, const double (&acc)[4][2][2],
                                        double alpha_eff) {
  using O = POrient<BM, BN, BK>;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int wm = warp % O::WM, wn = warp / O::WM;
  const int g = lane >> 2, q = lane & 3;
#pragma unroll
  for (int j = 0; j < 2; ++j)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int cc = t.n0 + wn * 16 + j * 8 + 2 * q + h;
      if (cc >= d.N) continue;
      double* cp = d.C + (size_t)cc * d.ldc;
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int r = t.m0 + wm * 32 + i * 8 + g;
        if (r < d.M) cp[r] = (alpha_eff == 1.0) ? acc[i][j][h] : alpha_eff * acc[i][j][h];
      }
    }
}

// DescFn(problem, GemmDesc&, int& wide) -> bool (problem present)
template <int BK, int STAGES, class DescFn>
__global__ void __launch_bounds__(kPThreads, 1) gemm_persistent_kernel(DescFn fn, int n_problems) {
  using Cfg = PCfg<BK, STAGES>;
  extern __shared__ __align__(16) double smem_p[];
  __shared__ GemmDesc s_desc[kPMaxProblems];
  __shared__ int s_cnt[kPMaxProblems];
  __shared__ int s_pref[kPMaxProblems + 1];
  __shared__ int s_tm[kPMaxProblems];
  __shared__ unsigned char s_wide[kPMaxProblems];

  if (threadIdx.x < n_problems) {
    const int p = threadIdx.x;
    GemmDesc d;
    int wide = 0, cnt = 0, tm = 1;
    if (fn(p, d, wide) && d.M > 0 && d.N > 0) {
      const int bm = wide ? 64 : 128, bn = wide ? 128 : 64;
      tm = (d.M + bm - 1) / bm;
      cnt = tm * ((d.N + bn - 1) / bn);
      s_desc[p] = d;
    }
    s_cnt[p] = cnt; s_tm[p] = tm; s_wide[p] = (unsigned char)wide;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int run = 0;
    for (int p = 0; p < n_problems; ++p) { s_pref[p] = run; run += s_cnt[p]; }
    s_pref[n_problems] = run;
  }
  __syncthreads();
  const int total = s_pref[n_problems];

  auto locate = [&](int tile) {
    PTileRef t;
    int p = 0;
    while (s_pref[p + 1] <= tile) ++p;       // <= 64 problems
    t.p = p;
    const int local = tile - s_pref[p], tm = s_tm[p];
    const int bm = s_wide[p] ? 64 : 128, bn = s_wide[p] ? 128 : 64;
    t.m0 = (local % tm) * bm; t.n0 = (local / tm) * bn;
    t.nk = (s_desc[p].K + BK - 1) / BK;
    if (t.nk < 1) t.nk = 1;
    return t;
  };

  int tile = blockIdx.x;
  if (tile >= total) return;
  PTileRef cur = locate(tile);

  // producer cursor: one k-step per call, STAGES-1 steps ahead of the consumer, across tiles
  PTileRef pt = cur;
  int ptile = tile, pk = 0, pstage = 0;
  auto produce = [&]() {
    if (ptile < total) {
      double* st = smem_p + pstage * Cfg::STAGE_DOUBLES;
      if (s_wide[pt.p]) p_load_step<64, 128, BK>(s_desc[pt.p], pt, pk, st);
      else p_load_step<128, 64, BK>(s_desc[pt.p], pt, pk, st);
      if (++pk == pt.nk) {
        ptile += gridDim.x;
        pk = 0;
        if (ptile < total) pt = locate(ptile);
      }
    }
    cp_async_commit();
    pstage = (pstage + 1 == STAGES) ? 0 : pstage + 1;
  };
#pragma unroll 1
  for (int s = 0; s < STAGES - 1; ++s) produce();

  double acc[4][2][2], pre[4][2][2];
  if (s_wide[cur.p]) p_fetch_c0<64, 128, BK>(s_desc[cur.p], cur, acc);
  else p_fetch_c0<128, 64, BK>(s_desc[cur.p], cur, acc);
  int cstage = 0;

  while (true) {
    const GemmDesc& d = s_desc[cur.p];
    const bool wide = s_wide[cur.p] != 0;
    const double alpha = d.alpha, beta = d.beta;
    const bool negA = (alpha == -1.0 && beta == 1.0);
    const double alpha_eff = negA ? 1.0 : alpha;
    const int sign_flip = negA ? (int)0x80000000 : 0;
    if (beta != 0.0) {
      const double bscale = beta / alpha_eff;
      if (bscale != 1.0) {
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 2; ++j) { acc[i][j][0] *= bscale; acc[i][j][1] *= bscale; }
      }
    }
    const int next_tile = tile + gridDim.x;
    const bool has_next = next_tile < total;
    PTileRef nxt = cur;
    if (has_next) nxt = locate(next_tile);
    const int pf_at = cur.nk > 3 ? cur.nk - 3 : 0;
#pragma unroll 1
    for (int k = 0; k < cur.nk; ++k) {
      cp_async_wait<STAGES - 2>();
      __syncthreads();
      produce();
      if (has_next && k == pf_at) {
        if (s_wide[nxt.p]) p_fetch_c0<64, 128, BK>(s_desc[nxt.p], nxt, pre);
        else p_fetch_c0<128, 64, BK>(s_desc[nxt.p], nxt, pre);
      }
      const double* cs = smem_p + cstage * Cfg::STAGE_DOUBLES;
      if (wide) p_compute_step<64, 128, BK>(cs, acc, sign_flip);
      else p_compute_step<128, 64, BK>(cs, acc, sign_flip);
      cstage = (cstage + 1 == STAGES) ? 0 : cstage + 1;
    }
    if (wide) p_store<64, 128, BK>(d, cur, acc, alpha_eff);
    else p_store<128, 64, BK>(d, cur, acc, alpha_eff);
    if (!has_next) break;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 2; ++j) { acc[i][j][0] = pre[i][j][0]; acc[i][j][1] = pre[i][j][1]; }
    cur = nxt;
    tile = next_tile;
  }
  cp_async_wait<0>();
}

}  // namespace ctaux
