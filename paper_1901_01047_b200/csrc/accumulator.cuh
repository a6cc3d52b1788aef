// S6: single-particle accumulation of CT-AUX on the device ("move the CT-AUX
// accumulator to the GPU").
//
//   PAPER.md:212  M is computed from a vertex configuration and its N_sigma; its Fourier coefficients are accumulated.
//   Eq. (28) PAPER.md:214  <G(k,iw_n)> = G0 - (1/beta) G0 <M(k,iw_n)> G0;   Eq. (29): Sigma = G0^-1 - <G>^-1.
//   Eq. (30)-(31) PAPER.md:232-238  delayed non-equispaced FFT: every sample is convolved with a localised
//   beta-periodic kernel phi onto an equispaced grid of L = m N_w points, the GRID is accumulated over the run, and ONE
//   transform at the end, divided by phi_w, gives the Fourier coefficients; phi is evaluated from a low-order polynomial.
//
// Readings (R1-R6):  M_sigma[j,l] = (E_j - 1) N_sigma[j,l]  (factor on the row; G_c = G0 - G0 M G0);
//   samples f = sign * M[j,l] at time tau_j - tau_l (folded to [0, beta) with the fermionic sign) and displacement
//   r_j - r_l;  Gaussian window exp(-(t/(s Delta))^2), s^2 = (2 sigma/(2 sigma - 1)) (w/pi), sigma = m/2, truncated
//   at w cells, tabulated with its derivative at kAccTab points per cell (cubic Hermite);  accumulators
//   grid[spin][r][l] are shared by all walkers of the context (the Monte-Carlo average sums over them anyway).
//
// Kernel shape: one CTA per (displacement r, walker, spin).  The vertices are bucketed by site first, so the pairs
// (j, l) with r_j - r_l = r are the products bucket(a) x bucket(a - r).  Every warp owns a PRIVATE copy of the tau grid
// of this r in shared memory and handles one sample at a time with one lane per touched grid point (2w <= 32): no
// atomics and no bank conflicts inside the spreading loop; the copies are summed and added to the global grid with
// L atomics per CTA.  HBM traffic: one 8-byte gather per element of N (sector-granular: 32 k^2 bytes per matrix).
#pragma once
#include "walker_state.cuh"

namespace ctaux {

constexpr int kAccTab = 32;       // window table points per grid cell
constexpr int kAccThreads = 256;  // 8 warps

struct AccCtx {
  int n_omega, m, w, L;        // positive frequencies, oversampling, window half-width (cells), grid points = m * n_omega
  int copies;                  // private grid copies per CTA (<= 8 warps)
  double inv_delta;            // L / beta
  double* grid;                // [2][Nc][L]
  const double* tab;           // [w*kAccTab + 1] window, then [w*kAccTab + 1] derivative * (1/kAccTab)
  const double* phi_hat;       // [n_omega]
  double* sign_sum;            // [1]
  long long* n_meas;           // [1]
  int32_t* site_start;         // [B][2][Nc + 1]   buckets per spin sector (the two sectors may see different sites)
  int32_t* site_list;          // [B][2][max_k]
  double* out;                 // [2][Nc][n_omega][2]  finalised coefficients (re, im)
};

// bucket the vertices of every (walker, spin sector) by the site that sector sees (counting sort; list order inside a bucket)
__global__ void __launch_bounds__(256) k_acc_bucket(DevCtx c, AccCtx a) {
  extern __shared__ int s_cnt[];   // [Nc + 1]
  const int w = blockIdx.x >> 1, sp = blockIdx.x & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  const int32_t* pair = c.cfg_site + c.cfg_off(w, st.cfg_cur);
  for (int i = threadIdx.x; i <= c.Nc; i += blockDim.x) s_cnt[i] = 0;
  __syncthreads();
  for (int i = threadIdx.x; i < k; i += blockDim.x) atomicAdd(&s_cnt[c.site(sp, pair[i]) + 1], 1);
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 0; i < c.Nc; ++i) s_cnt[i + 1] += s_cnt[i];
  }
  __syncthreads();
  int32_t* start = a.site_start + (size_t)blockIdx.x * (c.Nc + 1);
  for (int i = threadIdx.x; i <= c.Nc; i += blockDim.x) start[i] = s_cnt[i];
  // stable fill: one thread per site walks the list (k is a few thousand at most, Nc threads in parallel)
  int32_t* list = a.site_list + (size_t)blockIdx.x * c.max_k;
  for (int sidx = threadIdx.x; sidx < c.Nc; sidx += blockDim.x) {
    int pos = s_cnt[sidx];
    for (int i = 0; i < k; ++i)
      if (c.site(sp, pair[i]) == sidx) list[pos++] = i;
  }
}

__global__ void k_acc_sign(DevCtx c, AccCtx a) {
  double s = 0.0;
  for (int w = 0; w < c.B; ++w) s += (double)c.ws[w].sign;
  *a.sign_sum += s;
  *a.n_meas += c.B;
}

__device__ __forceinline__ double acc_window(const double* tab, int w, double x) {   // phi at |x| <= w cells
  x = fabs(x);
  const double u = x * kAccTab;
  int i = (int)u;
  if (i > w * kAccTab - 1) i = w * kAccTab - 1;
  const double f = u - (double)i;
  const double* d = tab + (w * kAccTab + 1);
  const double p0 = tab[i], p1 = tab[i + 1], d0 = d[i], d1 = d[i + 1];
  const double f2 = f * f, f3 = f2 * f;
  return (2.0 * f3 - 3.0 * f2 + 1.0) * p0 + (f3 - 2.0 * f2 + f) * d0 + (-2.0 * f3 + 3.0 * f2) * p1 + (f3 - f2) * d1;
}

__global__ void __launch_bounds__(kAccThreads) k_accumulate(DevCtx c, AccCtx a) {
  extern __shared__ __align__(16) double s_acc[];   // [copies][L] private grids, then the window table
  const int r = blockIdx.x, prob = blockIdx.y, wk = prob >> 1, sp = prob & 1;
  const WalkerState& st = c.ws[wk];
  const int k = st.k;
  if (k == 0) return;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int L = a.L, w = a.w, ntab = 2 * (w * kAccTab + 1);
  double* s_tab = s_acc + (size_t)a.copies * L;
  for (int i = tid; i < a.copies * L; i += kAccThreads) s_acc[i] = 0.0;
  for (int i = tid; i < ntab; i += kAccThreads) s_tab[i] = a.tab[i];
  __syncthreads();
  const size_t off = c.cfg_off(wk, st.cfg_cur);
  const double* tau = c.cfg_tau + off;
  const int32_t* spin = c.cfg_spin + off;
  const double* N = c.N(wk, sp, st.n_cur);
  const int32_t* pair = c.cfg_site + off;
  const int32_t* start = a.site_start + (size_t)prob * (c.Nc + 1);
  const int32_t* list = a.site_list + (size_t)prob * c.max_k;
  const double sgn_w = (double)st.sign;
  const int rx = r % c.Lx, ry = r / c.Lx;
  if (warp < a.copies) {
    double* mine = s_acc + (size_t)warp * L;
    for (int sa = 0; sa < c.Nc; ++sa) {
      // r_j - r_l = r with r_j = site sa  =>  r_l = sa - r
      int bx = sa % c.Lx - rx; if (bx < 0) bx += c.Lx;
      int by = sa / c.Lx - ry; if (by < 0) by += c.Ly;
      const int sb = bx + c.Lx * by;
      const int a0 = start[sa], ca = start[sa + 1] - a0, b0 = start[sb], cb = start[sb + 1] - b0;
      const int npair = ca * cb;
      for (int base = warp * 32; base < npair; base += a.copies * 32) {
        // every lane prepares one sample of this chunk ...
        double x = 0.0, val = 0.0;
        int l0 = 0;
        const int p = base + lane;
        if (p < npair) {
          const int j = list[a0 + p / cb], l = list[b0 + p % cb];
          double t = tau[j] - tau[l];
          double sg = sgn_w;
          if (t < 0.0) { sg = -sg; t += c.beta; }
          x = t * a.inv_delta;
          l0 = (int)floor(x);
          val = sg * (c.E(sp, spin[j], pair[j]) - 1.0) * N[(size_t)l * c.ld + j];
        }
        const int cnt = npair - base < 32 ? npair - base : 32;
        // ... and the warp spreads them one at a time, one lane per touched grid point
        for (int q = 0; q < cnt; ++q) {
          const double xq = __shfl_sync(0xffffffffu, x, q), vq = __shfl_sync(0xffffffffu, val, q);
          const int lq = __shfl_sync(0xffffffffu, l0, q);
          if (lane < 2 * w) {
            int gl = lq - w + 1 + lane;
            const double wgt = acc_window(s_tab, w, xq - (double)gl);
            double v = vq * wgt;
            if (gl < 0) { gl += L; v = -v; } else if (gl >= L) { gl -= L; v = -v; }   // beta-antiperiodic grid
            mine[gl] += v;
          }
          __syncwarp();
        }
      }
    }
  }
  __syncthreads();
  double* g = a.grid + ((size_t)sp * c.Nc + r) * L;
  for (int i = tid; i < L; i += kAccThreads) {
    double s = 0.0;
    for (int cp = 0; cp < a.copies; ++cp) s += s_acc[(size_t)cp * L + i];
    if (s != 0.0) atomicAdd(g + i, s);
  }
}

// End of the run: the length-L transform at the N_w positive fermionic frequencies, divided by phi_w (Eq. (31)):
//   out[sp][r][n] = (1/phi_n) sum_l grid[sp][r][l] e^{i (2n+1) pi l / L}
__global__ void __launch_bounds__(128) k_acc_finalize(DevCtx c, AccCtx a) {
  const int r = blockIdx.x, sp = blockIdx.y;
  const double* g = a.grid + ((size_t)sp * c.Nc + r) * a.L;
  const int twoL = 2 * a.L;
  for (int n = threadIdx.x; n < a.n_omega; n += blockDim.x) {
    double re = 0.0, im = 0.0;
    const int step = (2 * n + 1) % twoL;
    int ph = 0;                       // (2n+1) l mod 2L: the phase is pi * ph / L, reduced exactly in integers
    for (int l = 0; l < a.L; ++l) {
      double sn, cs;
      sincospi((double)ph / (double)a.L, &sn, &cs);
      const double v = g[l];
      re += v * cs; im += v * sn;
      ph += step; if (ph >= twoL) ph -= twoL;
    }
    const double inv = 1.0 / a.phi_hat[n];
    double* o = a.out + (((size_t)sp * c.Nc + r) * a.n_omega + n) * 2;
    o[0] = re * inv; o[1] = im * inv;
  }
}

}  // namespace ctaux
