// Grouped FP64 GEMM on the sm_100a FP64 tensor pipe (mma.sync m8n8k4 -> SASS DMMA.8x8x4) with the operand tiles
// staged by TMA (cp.async.bulk.tensor -> SASS UTMALDG) into shared memory and tracked by mbarriers.
//
// Serves S2 (candidate rows / columns), S4 (the rank-r flush with its compaction gather) and S5 (trailing updates of
// the blocked LU).  PAPER.md:226 ("rank-k_s operation"), PAPER.md:373 ("large matrix-matrix multiplications");
// BASELINE.json north_star: "hand-written sm_100a FP64 tensor-core (DMMA) GEMM tiles staged with TMA".
//
//   C[i,j] = beta * C0[rowmap[i], colmap[j]] + alpha * sum_k A[i,k] * B[k,j]          (all column-major, FP64)
//
// FP64 has no tcgen05.mma kind, so the math stays on mma.sync m8n8k4 with register accumulators; what TMA removes is
// the per-thread address arithmetic, bounds predicates and cp.async issue of the operand tiles (the instruction-heavy
// prologue that dominated the short-K flush tiles): ONE thread issues two bulk tensor copies per pipeline stage.
//
// Shared-memory layouts are chosen through the SHAPE OF THE TENSOR MAP so that the DMMA fragment loads (thread
// (g = lane/4, q = lane%4) reads A[row g][k q] and B[k q][col g]) are bank-conflict free without padding.  A 64-bit
// shared load is served per HALF-warp (g in 0..3 or 4..7, q in 0..3), so the 16 (g, q) pairs of a half-warp must fall
// into 16 different 8-byte bank pairs, i.e. the word index must be 4q + g%4 (or 4(g%4) + q) modulo 16:
//
//   * "M-major" operand, element (m, k) at base + m + k*ld (A of every GEMM here; B when its n index is contiguous):
//     viewed as a rank-3 tensor (4, K, M/4) with strides (8 B, ld*8 B, 32 B) and box (4, BK, 64/4): the tile lands as
//     [m/4][k][m%4], word index ((m/4)*BK + k)*4 + m%4  ==  4q + g%4  (mod 16).
//   * "K-major" operand, element (k, n) at base + k + n*ld (N as the right factor of the candidate-row GEMM, the U12
//     panel of the LU): rank-3 tensor (4, N, K/4) with strides (8 B, ld*8 B, 32 B) and box (4, 64, BK/4): the tile lands
//     as [k/4][n][k%4], word index ((k/4)*64 + n)*4 + k%4  ==  4(g%4) + q  (mod 16).
//   (The wider boxes one would like for the TMA engine -- [m/8][k][8], or 128-byte rows with the 128B swizzle --
//   were measured first: correct, but every fragment load is a 2-way bank conflict; ncu: 1.8 M conflicts per launch.)
//
// K tails: the tensor maps describe the CAPACITY of each buffer, not the live size of the walker's matrices, so
// elements with k >= K hold stale (finite or not) data: the fragments of the last k-chunk are masked in registers.
// M / N tails: rows / columns beyond the problem are computed from whatever the box holds and never stored.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "gemm_dmma.cuh"

namespace ctaux {

struct TmaGemmDesc {
  int M, N, K;
  const CUtensorMap* tmA; int a_m0, a_k0;   // M-major view: tile (m0, k0) at coordinates (0, a_k0 + k0, (a_m0 + m0) / 4)
  const CUtensorMap* tmB; int b_k0, b_n0;   // N-major view: (0, b_k0 + k0, (b_n0 + n0) / 4);  K-major: (0, b_n0 + n0, (b_k0 + k0) / 4)
  double* C; int ldc;
  const double* C0; int ldc0;               // source of the beta term (may alias C when no maps are given)
  const int* rowmap;                        // nullptr = identity
  const int* colmap;
  double alpha, beta;
};

// ---- mbarrier / TMA primitives (PTX ISA: mbarrier, cp.async.bulk.tensor)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, int c0, int c1, int c2, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];\n"
               ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* tm, int c0, int c1, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n"
               ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* tm) {
  asm volatile("prefetch.tensormap [%0];\n" ::"l"(tm) : "memory");
}

// ---- distributed shared memory: data + signal in one message (st.async onto the receiver's mbarrier)
// shared::cluster address of `addr` (a shared::cta address of this CTA) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
// two doubles into a peer CTA's shared memory; completes 16 bytes of transaction on the PEER's mbarrier
__device__ __forceinline__ void st_async_2f64(uint32_t dst_cluster_addr, double a, double b, uint32_t mbar_cluster_addr) {
  asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];\n"
               ::"r"(dst_cluster_addr), "d"(a), "d"(b), "r"(mbar_cluster_addr) : "memory");
}
// one double into a CTA of the cluster; completes 8 bytes of transaction on that CTA's mbarrier
__device__ __forceinline__ void st_async_f64(uint32_t dst_cluster_addr, double a, uint32_t mbar_cluster_addr) {
  asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];\n"
               ::"r"(dst_cluster_addr), "l"(__double_as_longlong(a)), "r"(mbar_cluster_addr) : "memory");
}

constexpr int kTmaBM = 64, kTmaBN = 64, kTmaBK = 16;
constexpr int kTmaThreads = 128;   // 4 warps, 32 x 32 warp tiles (2 x 2)

template <int STAGES>
struct TmaCfg {
  static constexpr int A_STAGE = kTmaBM * kTmaBK;   // doubles
  static constexpr int B_STAGE = kTmaBN * kTmaBK;
  static constexpr int STAGE_BYTES = (A_STAGE + B_STAGE) * 8;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024;   // + slack to align the ring to 1024 B
};

// One CTA computes one 64 x 64 tile.  `it` counts the k-chunks this CTA has pushed through the ring so far (stage
// and mbarrier parity follow from it); the caller guarantees that every thread has passed a __syncthreads() since the
// ring was last read (tile loop below).
template <int STAGES, bool B_KMAJOR, bool PRE>
__device__ __forceinline__ void tma_gemm_tile(const TmaGemmDesc& d, int tile_m, int tile_n, double* ring, uint64_t* full,
                                              uint32_t& it, const int* pre_srow = nullptr, const int* pre_scol = nullptr) {
  using Cfg = TmaCfg<STAGES>;
  constexpr int BK = kTmaBK, TM = 4, TN = 4;
  const int tid = threadIdx.x;
  const int warp = tid >> 5, lane = tid & 31;
  const int wm = warp & 1, wn = warp >> 1;
  const int g = lane >> 2, q = lane & 3;
  const int m0 = tile_m * kTmaBM, n0 = tile_n * kTmaBN;
  const int M = d.M, N = d.N, K = d.K;
  const int nk = (K + BK - 1) / BK;

  auto issue = [&](int kt) {   // thread 0 only
    const uint32_t slot = (it + (uint32_t)kt) % STAGES;
    double* As = ring + (size_t)slot * (Cfg::A_STAGE + Cfg::B_STAGE);
    double* Bs = As + Cfg::A_STAGE;
    const int k0 = kt * BK;
    mbar_expect_tx(full + slot, (uint32_t)Cfg::STAGE_BYTES);
    tma_load_3d(As, d.tmA, 0, d.a_k0 + k0, (d.a_m0 + m0) >> 2, full + slot);
    if (B_KMAJOR) tma_load_3d(Bs, d.tmB, 0, d.b_n0 + n0, (d.b_k0 + k0) >> 2, full + slot);
    else tma_load_3d(Bs, d.tmB, 0, d.b_k0 + k0, (d.b_n0 + n0) >> 2, full + slot);
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s)
      if (s < nk) issue(s);
  }

  // index maps of this thread's fragment rows / columns (C0 gather = compaction of the flush)
  int crow[TM], srow[TM], ccol[TN][2], scol[TN][2];
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    crow[i] = m0 + wm * 32 + i * 8 + g;
    if (PRE) srow[i] = pre_srow[i];
    else srow[i] = (d.rowmap && crow[i] < M) ? d.rowmap[crow[i]] : crow[i];
  }
#pragma unroll
  for (int j = 0; j < TN; ++j)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      ccol[j][h] = n0 + wn * 32 + j * 8 + 2 * q + h;
      if (PRE) scol[j][h] = pre_scol[j * 2 + h];
      else scol[j][h] = (d.colmap && ccol[j][h] < N) ? d.colmap[ccol[j][h]] : ccol[j][h];
    }

  // Accumulators start from C0[gather] (scaled by beta/alpha when that is not 1): the loads are in flight while the
  // ring fills and the epilogue is a pure store.  The in-place update C = C0 - A*B (alpha = -1, beta = 1: flush, LU
  // trailing updates) flips the sign bit of the A fragments instead.
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
    const uint32_t cur = it + (uint32_t)kt;
    const uint32_t slot = cur % STAGES;
    mbar_wait(full + slot, (cur / STAGES) & 1u);
    __syncthreads();   // every warp is done with chunk kt-1: its slot may be refilled
    if (tid == 0 && kt + STAGES - 1 < nk) issue(kt + STAGES - 1);
    const double* a_s = ring + (size_t)slot * (Cfg::A_STAGE + Cfg::B_STAGE) + (wm * 8 + (g >> 2)) * (BK * 4) + (g & 3);
    const double* b_s = ring + (size_t)slot * (Cfg::A_STAGE + Cfg::B_STAGE) + Cfg::A_STAGE;
    const int kv = K - kt * BK;   // valid k values in this chunk (>= BK except in the last one)
    if (kv >= BK) {
#pragma unroll
      for (int k4 = 0; k4 < BK; k4 += 4) {
        double af[TM], bf[TN];
#pragma unroll
        for (int i = 0; i < TM; ++i) {
          const double a = a_s[i * (2 * BK * 4) + (k4 + q) * 4];
          af[i] = __hiloint2double(__double2hiint(a) ^ sign_flip, __double2loint(a));
        }
#pragma unroll
        for (int j = 0; j < TN; ++j) {
          if (B_KMAJOR) bf[j] = b_s[((k4 >> 2) * kTmaBN + wn * 32 + j * 8 + g) * 4 + q];
          else bf[j] = b_s[((wn * 8 + j * 2 + (g >> 2)) * BK + k4 + q) * 4 + (g & 3)];
        }
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
          for (int j = 0; j < TN; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
      }
    } else {   // K tail: the boxes hold stale data beyond K, masked in registers
      for (int k4 = 0; k4 < kv; k4 += 4) {
        const bool dead = k4 + q >= kv;
        double af[TM], bf[TN];
#pragma unroll
        for (int i = 0; i < TM; ++i) {
          const double a = a_s[i * (2 * BK * 4) + (k4 + q) * 4];
          af[i] = dead ? 0.0 : __hiloint2double(__double2hiint(a) ^ sign_flip, __double2loint(a));
        }
#pragma unroll
        for (int j = 0; j < TN; ++j) {
          double b;
          if (B_KMAJOR) b = b_s[((k4 >> 2) * kTmaBN + wn * 32 + j * 8 + g) * 4 + q];
          else b = b_s[((wn * 8 + j * 2 + (g >> 2)) * BK + k4 + q) * 4 + (g & 3)];
          bf[j] = dead ? 0.0 : b;
        }
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
          for (int j = 0; j < TN; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
      }
    }
  }
  it += (uint32_t)nk;

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

__device__ __forceinline__ double* tma_ring_base(double* raw) {
  return reinterpret_cast<double*>((reinterpret_cast<uintptr_t>(raw) + 1023) & ~(uintptr_t)1023);
}

// Grouped launch: blockIdx.y = problem, the CTAs of a problem stride over its tiles (a stale host-side tile count
// costs balance, never correctness).  DescFn(problem, TmaGemmDesc&) -> bool, evaluated on the device.
template <int STAGES, bool B_KMAJOR, int MINB, class DescFn>
__global__ void __launch_bounds__(kTmaThreads, MINB) gemm_tma_kernel(DescFn fn) {
  extern __shared__ __align__(16) double smem_tma_raw[];
  __shared__ uint64_t full[STAGES];
  double* ring = tma_ring_base(smem_tma_raw);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) mbar_init(full + s, 1);
    mbar_fence_init();
  }
  TmaGemmDesc d;
  const bool live = fn(blockIdx.y, d) && d.M > 0 && d.N > 0;
  __syncthreads();
  if (!live) return;
  const int tm = (d.M + kTmaBM - 1) / kTmaBM, tn = (d.N + kTmaBN - 1) / kTmaBN;
  uint32_t it = 0;
  for (int t = blockIdx.x; t < tm * tn; t += gridDim.x) {
    tma_gemm_tile<STAGES, B_KMAJOR, false>(d, t % tm, t / tm, ring, full, it);
    __syncthreads();
  }
}

// Flush form (S4): the tile -> (tile_m, tile_n) mapping of the FIRST tile of every CTA uses a host-side tile count
// `tmax`, so the loads of its compaction-map entries (map of problem p at maps + (p >> 1) * map_stride, rows and
// columns alike) are issued BEFORE the device-side descriptor has arrived.  Tiles the grid does not cover (stale
// hint) are strided over afterwards.  Speculative map reads are clamped to the walker's own map.
template <int STAGES, int MINB, class DescFn>
__global__ void __launch_bounds__(kTmaThreads, MINB)
    gemm_tma_flush_kernel(DescFn fn, const int* maps, int map_stride, int tmax) {
  extern __shared__ __align__(16) double smem_tma_raw[];
  __shared__ uint64_t full[STAGES];
  double* ring = tma_ring_base(smem_tma_raw);
  const int tile_m = blockIdx.x % tmax, tile_n = blockIdx.x / tmax;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int wm = warp & 1, wn = warp >> 1, g = lane >> 2, q = lane & 3;
  const int* map = maps + (size_t)(blockIdx.y >> 1) * map_stride;
  int psrow[4], pscol[8];
#pragma unroll
  for (int i = 0; i < 4; ++i) psrow[i] = __ldg(map + min(tile_m * kTmaBM + wm * 32 + i * 8 + g, map_stride - 1));
#pragma unroll
  for (int j = 0; j < 4; ++j)
#pragma unroll
    for (int h = 0; h < 2; ++h) pscol[j * 2 + h] = __ldg(map + min(tile_n * kTmaBN + wn * 32 + j * 8 + 2 * q + h, map_stride - 1));
  if (threadIdx.x == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) mbar_init(full + s, 1);
    mbar_fence_init();
  }
  TmaGemmDesc d;
  const bool live = fn(blockIdx.y, d) && d.M > 0 && d.N > 0;
  __syncthreads();
  if (!live) return;
  uint32_t it = 0;
  if (tile_m * kTmaBM < d.M && tile_n * kTmaBN < d.N) {
    tma_gemm_tile<STAGES, false, true>(d, tile_m, tile_n, ring, full, it, psrow, pscol);
  }
  const int tm = (d.M + kTmaBM - 1) / kTmaBM, tn = (d.N + kTmaBN - 1) / kTmaBN;
  if (tm <= tmax && tn <= tmax) return;
  const int rows_x = tm > tmax ? tm - tmax : 0, cols_x = tn > tmax ? tn - tmax : 0;
  const int tm_cov = tm < tmax ? tm : tmax;
  const int extra = rows_x * tn + tm_cov * cols_x;
  for (int e = blockIdx.x; e < extra; e += gridDim.x) {
    int em, en;
    if (e < rows_x * tn) { em = tmax + e % rows_x; en = e / rows_x; }
    else { const int f = e - rows_x * tn; em = f % tm_cov; en = tmax + f / tm_cov; }
    __syncthreads();
    tma_gemm_tile<STAGES, false, false>(d, em, en, ring, full, it);
  }
}


}  // namespace ctaux
