// Forward-error monitor of the incrementally updated N_sigma  (BASELINE.json north_star: "N within a relative
// Frobenius error of 1e-10", "periodic from-scratch rebuild").
//
// Fast updates of an inverse amplify the error N already carries: a column change A -> A' maps delta = N - A^-1 to
// (A'^-1 A) delta (A A'^-1), so the drift of a chain is data dependent (measured: 4e-11 ... 2e-10 after ONE sweep of
// config 4 from a thermalised start, for ANY way of inverting the small S matrix; tests/test_drift_model.py).  A fixed
// rebuild cadence therefore either wastes rebuilds or misses the bar; the library measures the error instead and
// rebuilds when it is needed.
//
//   delta = N - A^-1 = (N A - 1) A^-1  ~=  (N A - 1) N            (first order in delta)
//   Hutchinson: for a Rademacher vector z,  E |z^T M|^2 = |M|_F^2, hence with
//       y^T = z^T N,    t^T = y^T A - z^T,    d^T = t^T N :      |d|^2 ~ |delta|_F^2,   |y|^2 ~ |N|_F^2
//   and  est = sqrt( sum_p |d_p|^2 / sum_p |y_p|^2 )  over kProbes independent probes estimates the relative
//   Frobenius error of N -- the very quantity the parity bar is stated in.
//
// Cost per check and matrix: two passes over N (shared by the probes) and k^2 G0 interpolations (A is never stored).
// Every output element is ONE warp's dot product reduced in a fixed order: the estimate is deterministic.
#pragma once
#include "walker_state.cuh"

namespace ctaux {

constexpr int kProbes = 4;
constexpr int kMonWarps = 8;   // warps per CTA of the monitor kernels: one output column per warp

__device__ __forceinline__ double rademacher(uint32_t i, uint32_t p, uint32_t salt) {
  uint32_t h = i * 0x9E3779B1u ^ (p + 1u) * 0x85EBCA77u ^ salt * 0xC2B2AE3Du;
  h ^= h >> 15; h *= 0x2C1B3C6Du; h ^= h >> 12; h *= 0x297A2D39u; h ^= h >> 15;
  return (h & 0x10000u) ? 1.0 : -1.0;
}

// out[p][j] = sum_i w_p[i] N[i,j]  for the kProbes probes; w_p = Rademacher(i, p, salt) when `wbuf` is null.
// mon layout per problem (walker, spin): [3 vectors y, t, d][kProbes][ld].
__global__ void __launch_bounds__(kMonWarps * 32) k_mon_vecmat(DevCtx c, double* mon, int src, int dst, uint32_t salt) {
  const int prob = blockIdx.y, w = prob >> 1, sp = prob & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double* base = mon + (size_t)prob * 3 * kProbes * c.ld;
  const double* wbuf = src < 0 ? nullptr : base + (size_t)src * kProbes * c.ld;
  double* out = base + (size_t)dst * kProbes * c.ld;
  const double* N = c.N(w, sp, st.n_cur);
  for (int j = blockIdx.x * kMonWarps + warp; j < k; j += gridDim.x * kMonWarps) {
    const double* col = N + (size_t)j * c.ld;
    double acc[kProbes];
#pragma unroll
    for (int p = 0; p < kProbes; ++p) acc[p] = 0.0;
    for (int i = lane; i < k; i += 32) {
      const double v = col[i];
#pragma unroll
      for (int p = 0; p < kProbes; ++p) acc[p] += (wbuf ? wbuf[(size_t)p * c.ld + i] : rademacher((uint32_t)i, (uint32_t)p, salt)) * v;
    }
#pragma unroll
    for (int p = 0; p < kProbes; ++p) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc[p] += __shfl_xor_sync(0xffffffffu, acc[p], o);
      if (lane == 0) out[(size_t)p * c.ld + j] = acc[p];
    }
  }
}

// t[p][l] = sum_j y[p][j] A[j,l] - z_p[l],   A[j,l] = delta_jl E_l - g(j,l) (E_l - 1)   (Eq. (27))
__global__ void __launch_bounds__(kMonWarps * 32) k_mon_resid(DevCtx c, double* mon, uint32_t salt) {
  const int prob = blockIdx.y, w = prob >> 1, sp = prob & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double* base = mon + (size_t)prob * 3 * kProbes * c.ld;
  const double* y = base;
  double* t = base + (size_t)kProbes * c.ld;
  const size_t off = c.cfg_off(w, st.cfg_cur);
  const int32_t* site = c.cfg_site + off;
  const double* tau = c.cfg_tau + off;
  for (int l = blockIdx.x * kMonWarps + warp; l < k; l += gridDim.x * kMonWarps) {
    const double El = c.E(sp, c.cfg_spin[off + l], site[l]);
    const int sl = c.site(sp, site[l]);
    const double tl = tau[l];
    double acc[kProbes];
#pragma unroll
    for (int p = 0; p < kProbes; ++p) acc[p] = 0.0;
    for (int j = lane; j < k; j += 32) {
      const double a = (j == l) ? (El - c.g00 * (El - 1.0)) : -c.g(c.disp(c.site(sp, site[j]), sl), tau[j] - tl) * (El - 1.0);
#pragma unroll
      for (int p = 0; p < kProbes; ++p) acc[p] += y[(size_t)p * c.ld + j] * a;
    }
#pragma unroll
    for (int p = 0; p < kProbes; ++p) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc[p] += __shfl_xor_sync(0xffffffffu, acc[p], o);
      if (lane == 0) t[(size_t)p * c.ld + l] = acc[p] - rademacher((uint32_t)l, (uint32_t)p, salt);
    }
  }
}

// est[prob] = sqrt( sum_p |d_p|^2 / sum_p |y_p|^2 ), one CTA per problem, fixed summation order
__global__ void __launch_bounds__(256) k_mon_final(DevCtx c, const double* mon, double* est) {
  const int prob = blockIdx.x, w = prob >> 1;
  const int k = c.ws[w].k;
  const double* base = mon + (size_t)prob * 3 * kProbes * c.ld;
  const double* y = base;
  const double* d = base + (size_t)2 * kProbes * c.ld;
  __shared__ double s_y[256], s_d[256];
  double ay = 0.0, ad = 0.0;
  for (int p = 0; p < kProbes; ++p)
    for (int j = threadIdx.x; j < k; j += 256) {
      const double vy = y[(size_t)p * c.ld + j], vd = d[(size_t)p * c.ld + j];
      ay += vy * vy; ad += vd * vd;
    }
  s_y[threadIdx.x] = ay; s_d[threadIdx.x] = ad;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) { s_y[threadIdx.x] += s_y[threadIdx.x + o]; s_d[threadIdx.x] += s_d[threadIdx.x + o]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double e = (k > 0 && s_y[0] > 0.0) ? sqrt(s_d[0] / s_y[0]) : 0.0;
    if (!(e == e)) e = 1e300;   // NaN: certainly rebuild
    est[prob] = e;
  }
}

}  // namespace ctaux
