// Bare cluster propagator of the DCA on the device: the G0(r, tau) table the walker consumes,
// from the cluster self-energy instead of the isolated-cluster closed form.
//
//   Eq. (6)-(8) PAPER.md:85-93   Gbar(K, iw_n) = (Nc/V_BZ) int dk phi_K(k) [i w_n - eps_k + mu - Sigma_c(K, iw_n)]^-1
//   Eq. (9)     PAPER.md:97      cluster exclusion  G0c(K, iw_n) = [Gbar^-1 + Sigma_c]^-1
//   Eq. (45)    PAPER.md:517     eps_k = -2t (cos kx + cos ky)
// Readings G1-G4: standard square patches with an n_quad x n_quad midpoint rule; G0c(r) = (1/Nc) sum_K
// e^{iK.r} G0c(K); Matsubara sum over +-n from the N_w positive frequencies with the tail
// 1/(iw) + <eps-mu>/(iw)^2 + <(eps-mu)^2>/(iw)^3 summed analytically; table T[d][m], m = 0..M, end points one-sided.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ctaux {

struct G0Ctx {
  int Lx, Ly, Nc, n_omega, n_quad, n_tau;
  double t, mu, beta;
  const double* sigma;   // [Nc][n_omega][2] or null
  double* remK;          // [Nc][n_omega][2]  G0c(K, iw_n) minus its three-moment tail
  double* mom;           // [Nc][2]           <eps - mu>, <(eps - mu)^2> per patch
  double* remR;          // [Nc][n_omega][2]  the same in r
  double* momR;          // [Nc][2]
  double* table;         // [Nc][n_tau + 1]
};

// one CTA per cluster momentum K: patch quadrature for every frequency, cluster exclusion, tail removal
__global__ void __launch_bounds__(256) k_g0_coarse(G0Ctx c) {
  const int K = blockIdx.x, kx = K % c.Lx, ky = K / c.Lx;
  const double Kx = 2.0 * M_PI * kx / c.Lx, Ky = 2.0 * M_PI * ky / c.Ly;
  const int nq = c.n_quad, nq2 = nq * nq;
  extern __shared__ double s_eps[];   // [nq2] eps on the patch
  for (int p = threadIdx.x; p < nq2; p += blockDim.x) {
    const double ox = ((p % nq + 0.5) / nq - 0.5) * (2.0 * M_PI / c.Lx);
    const double oy = ((p / nq + 0.5) / nq - 0.5) * (2.0 * M_PI / c.Ly);
    s_eps[p] = -2.0 * c.t * (cos(Kx + ox) + cos(Ky + oy));
  }
  __syncthreads();
  // patch moments, summed in a fixed order by every thread (nq2 is small)
  double m1 = 0.0, m2 = 0.0;
  for (int p = 0; p < nq2; ++p) { const double x = s_eps[p] - c.mu; m1 += x; m2 += x * x; }
  m1 /= nq2; m2 /= nq2;
  if (threadIdx.x == 0) { c.mom[2 * K] = m1; c.mom[2 * K + 1] = m2; }
  for (int n = threadIdx.x; n < c.n_omega; n += blockDim.x) {
    const double wn = (2 * n + 1) * M_PI / c.beta;
    const double sr = c.sigma ? c.sigma[((size_t)K * c.n_omega + n) * 2] : 0.0;
    const double si = c.sigma ? c.sigma[((size_t)K * c.n_omega + n) * 2 + 1] : 0.0;
    double gr = 0.0, gi = 0.0;
    for (int p = 0; p < nq2; ++p) {           // 1 / (i wn - eps + mu - Sigma) = conj(z) / |z|^2
      const double zr = -s_eps[p] + c.mu - sr, zi = wn - si;
      const double inv = 1.0 / (zr * zr + zi * zi);
      gr += zr * inv; gi -= zi * inv;
    }
    gr /= nq2; gi /= nq2;                     // Gbar, Eq. (7)
    // Eq. (9): G0c = 1 / (1/Gbar + Sigma)
    const double d = 1.0 / (gr * gr + gi * gi);
    const double ir = gr * d + sr, ii = -gi * d + si;
    const double e = 1.0 / (ir * ir + ii * ii);
    double g0r = ir * e, g0i = -ii * e;
    // tail: 1/(iw) = -i/w,  1/(iw)^2 = -1/w^2,  1/(iw)^3 = i/w^3
    g0r -= -m1 / (wn * wn);
    g0i -= -1.0 / wn + m2 / (wn * wn * wn);
    c.remK[((size_t)K * c.n_omega + n) * 2] = g0r;
    c.remK[((size_t)K * c.n_omega + n) * 2 + 1] = g0i;
  }
}

// K -> r (reading G2): remR[d][n] = (1/Nc) sum_K e^{iK.r_d} remK[K][n];  moments likewise (real by inversion symmetry)
__global__ void __launch_bounds__(256) k_g0_to_r(G0Ctx c) {
  const int d = blockIdx.x, rx = d % c.Lx, ry = d / c.Lx;
  for (int n = threadIdx.x; n < c.n_omega + 1; n += blockDim.x) {
    double ar = 0.0, ai = 0.0;
    for (int K = 0; K < c.Nc; ++K) {
      double sn, cs;
      // K.r = 2 pi (kx rx / Lx + ky ry / Ly): reduced exactly in integers before the sincos
      const int num = ((K % c.Lx) * rx * c.Ly + (K / c.Lx) * ry * c.Lx) % (c.Lx * c.Ly);
      sincospi(2.0 * num / (double)(c.Lx * c.Ly), &sn, &cs);
      if (n < c.n_omega) {
        const double vr = c.remK[((size_t)K * c.n_omega + n) * 2], vi = c.remK[((size_t)K * c.n_omega + n) * 2 + 1];
        ar += cs * vr - sn * vi; ai += cs * vi + sn * vr;
      } else {
        ar += cs * c.mom[2 * K]; ai += cs * c.mom[2 * K + 1];   // (n == n_omega: the two moments ride along)
      }
    }
    if (n < c.n_omega) {
      c.remR[((size_t)d * c.n_omega + n) * 2] = ar / c.Nc;
      c.remR[((size_t)d * c.n_omega + n) * 2 + 1] = ai / c.Nc;
    } else {
      c.momR[2 * d] = ar / c.Nc; c.momR[2 * d + 1] = ai / c.Nc;
    }
  }
}

// iw_n -> tau (readings G3, G4): one warp per table entry, lanes stride over the frequencies, fixed reduction order
__global__ void __launch_bounds__(256) k_g0_to_tau(G0Ctx c) {
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  const int M = c.n_tau;
  if (warp >= c.Nc * (M + 1)) return;
  const int d = warp / (M + 1), m = warp % (M + 1);
  double acc = 0.0;
  for (int n = lane; n < c.n_omega; n += 32) {
    // w_n tau_m = (2n+1) pi m / M, reduced exactly modulo 2 pi in integers
    const long long num = ((long long)(2 * n + 1) * m) % (2LL * M);
    double sn, cs;
    sincospi((double)num / (double)M, &sn, &cs);
    const double fr = c.remR[((size_t)d * c.n_omega + n) * 2], fi = c.remR[((size_t)d * c.n_omega + n) * 2 + 1];
    acc += fr * cs + fi * sn;                 // Re[(fr + i fi)(cos - i sin)]
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) {
    const double tau = (m == M) ? c.beta : m * (c.beta / M);
    const double c1 = d == 0 ? 1.0 : 0.0, c2 = c.momR[2 * d], c3 = c.momR[2 * d + 1];
    c.table[(size_t)d * (M + 1) + m] = (2.0 / c.beta) * acc - 0.5 * c1 + c2 * (2.0 * tau - c.beta) / 4.0 + c3 * tau * (c.beta - tau) / 4.0;
  }
}

}  // namespace ctaux
