// Device-side state of the batched CT-AUX walkers and small device helpers
// (Philox4x32-10, G0 interpolation, E = e^{-gamma sigma s}).  SURVEY.md 8c.1 / DESIGN.md.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace ctaux {

constexpr int kMaxDelay = 256;
constexpr int kMaxSplitK = 8;

// TMA tensor maps of one (walker, spin): every buffer a GEMM reads as an operand, in the view its role needs
// (gemm_tma.cuh: "M-major" rank-3 view for left operands and n-contiguous right operands, "K-major" swizzled rank-2
// view for k-contiguous right operands).  Built once by ctaux_create; they describe capacities, not live sizes.
enum TmapId { TM_N0_M = 0, TM_N1_M, TM_N0_K, TM_N1_K, TM_BM_M, TM_UM_M, TM_UT_M, TM_V_N, TM_SINV_K, TM_GX_N, TM_T_K, TM_LINV_M, TM_COUNT };

struct LogEntry {  // == ctaux_log_entry
  uint64_t p;
  int32_t type, arg;
  double tau;
  int32_t spin, accepted;
  double R, u;
};

struct PropInfo {  // one pre-expanded proposal of the current window (16 bytes)
  uint32_t type_cand;  // bits 0-1: type (0 insert, 1 remove, 2 flip); bits 2..: candidate index (inserts)
  uint32_t w1;         // word used for the removal index
  double u;            // uniform for the Metropolis test
};

struct WalkerState {
  uint32_t key0, key1;
  int32_t k;        // expansion order at block start
  int32_t cfg_cur;  // current configuration buffer (0/1)
  int32_t n_cur;    // current N buffer (0/1), both spins
  int32_t n_src;    // N buffer the pending flush reads (== n_cur when r == 0)
  int32_t status;   // 0 ok, else CTAUX_E*
  int32_t sign;
  uint64_t next_id, p;
  int32_t sweeps_left, props_left;
  // current block
  int32_t m;       // insertion candidates pre-expanded
  int32_t win;     // proposals in the window
  int32_t r;       // accepted changes (rank of the flush)
  int32_t k_new;   // expansion order after the block
  int32_t active;  // 1 while the walker still has proposals to do in this sweep call
  int32_t pad0;
  // statistics
  int64_t acc_ins, acc_rem, sweeps, blocks, flushes, rebuilds, sum_rank, log_count, guard_ends, acc_flip;
  double flops_cand, flops_flush, flops_rebuild, min_margin, sum_k, flops_usinv, flops_cand_alg;
};

// Everything a kernel needs: passed by value (fits the 4 KB parameter space easily).
struct DevCtx {
  int B, Lx, Ly, Nc, M;
  int flips;   // 1: spin flip as a third move (ctaux_params.flip_moves)
  int max_k, mmax, winmax, delay;
  int cap;   // max_k + mmax : extended slots
  int ld;    // leading dimension of every N / Gx / U buffer (cap rounded up to 8)
  int ldm;   // leading dimension of Bm (mmax rounded up to 8)
  int ldr;   // leading dimension of Vt / Sinv in global memory (delay rounded up to 8)
  int log_capacity;
  double beta, K, tau_scale, g00;
  // Interacting pairs (Eq. (19)-(25)): H_int = sum_p U_p [n_{a_p up} n_{b_p dn} - ...]
  // over n_pairs = N_corr pairs.  A vertex is (pair, tau, s): cfg_site holds the PAIR index; the up matrix sees site
  // a_p, the down matrix site b_p, with gamma_p from Eq. (25).  The on-site Hubbard model is the identity table
  // (pair p = site p, N_corr = Nc, one gamma), so every kernel goes through these tables.
  int n_pairs;
  int onsite;                 // 1: the on-site model (identity tables): the accessors below answer from the four constants
  double egm, egp, iem_m, iem_p;   //    e^{-gamma}, e^{+gamma}, 1/(e^{-gamma} - 1), 1/(e^{+gamma} - 1) of that model
  const int32_t* pair_site;   // [2][n_pairs]  site of the up / down electron of pair p
  const double* pair_E;       // [2][n_pairs]  E for sigma*s = +1 (e^{-gamma_p}), then for sigma*s = -1 (e^{+gamma_p})
  const double* pair_iem1;    // [2][n_pairs]  1 / (E - 1) for the same two cases
  double guard_amp;  // rounding-amplification limit of the bordered ratio evaluation (k_propose)
  const double* table;  // [Nc][M+1]
  WalkerState* ws;      // [B]
  // configuration, double buffered, extended slots: [B][2][cap]
  int32_t* cfg_site; double* cfg_tau; int32_t* cfg_spin; uint64_t* cfg_id;
  PropInfo* prop;       // [B][winmax]
  double* Nbuf;         // [B][2 spins][2 bufs][ld*ld]
  double* Bm;           // [B][2][ldm*cap]   candidate rows  g(c,j)(E_j-1), m x k col-major
  double* gxC;          // [B][2][ld*ldm]    g_ext[:, C] per spin sector, stored n-contiguous: element (i, c) at i*ldm + c
  double* Gx;           // [B][2][ld*mmax]   N_ext * g_ext[:, C]
  double* Tbuf;         // [B][2][ld*ld]  A*N of the Newton-Schulz refresh (rebuild_mode 1), else null
  unsigned long long* resid;  // [B*2]  max |A N - 1| per matrix as the bit pattern of a non-negative double
  double* skbuf;        // [B][2][kMaxSplitK][skstride]  split-K partial products of the S2 GEMMs
  size_t skstride;      // max(ldm*cap, ld*mmax)
  double* Um;           // [B][2][ld*delay]  U = X[:, J]
  double* Ut;           // [B][2][ld*delay]  U * S^-1
  double* Vt;           // [B][2][ld*delay]  V = (rows J of N_ext)^T, k' x r col-major (n-contiguous right operand of the flush)
  double* Sinv;         // [B][2][ldr*delay]
  int32_t* J;           // [B][delay]
  int32_t* rowmap;      // [B][cap]  new list position -> extended slot
  LogEntry* log;        // [B][log_capacity]
  int32_t* n_active;    // [1] walkers still active (device), mirrored to pinned host
  // rebuild scratch
  double* colbuf;       // [B][2][ld]
  double* rowbuf;       // [B][2][ld]
  int32_t* perm;        // [B][2][ld]
  // tensor maps of the GEMM operand buffers [B][2][TM_COUNT] (gemm_tma.cuh)
  const CUtensorMap* tmaps;
  __device__ __forceinline__ const CUtensorMap* tm(int w, int s, int id) const { return tmaps + ((size_t)w * 2 + s) * TM_COUNT + id; }

  __device__ __forceinline__ size_t cfg_off(int w, int buf) const { return ((size_t)w * 2 + buf) * cap; }
  __device__ __forceinline__ double* N(int w, int s, int buf) const {
    return Nbuf + (((size_t)w * 2 + s) * 2 + buf) * (size_t)ld * ld;
  }
  // sigma = +1 for sidx 0 (up), -1 for sidx 1; E = exp(-gamma_p sigma s)
  __device__ __forceinline__ double E(int sidx, int s, int p) const {
    const bool minus = (sidx == 0) == (s > 0);
    if (onsite) return minus ? egm : egp;
    return __ldg(pair_E + (minus ? 0 : n_pairs) + p);
  }
  __device__ __forceinline__ double iem1(int sidx, int s, int p) const {   // 1 / (E - 1)
    const bool minus = (sidx == 0) == (s > 0);
    if (onsite) return minus ? iem_m : iem_p;
    return __ldg(pair_iem1 + (minus ? 0 : n_pairs) + p);
  }
  __device__ __forceinline__ int site(int sidx, int p) const { return onsite ? p : __ldg(pair_site + sidx * n_pairs + p); }
  // compile-time forms for the latency-critical S3 kernels (instantiated once per model class)
  template <bool ON> __device__ __forceinline__ double Et(int sidx, int s, int p) const {
    const bool minus = (sidx == 0) == (s > 0);
    if (ON) return minus ? egm : egp;
    return __ldg(pair_E + (minus ? 0 : n_pairs) + p);
  }
  template <bool ON> __device__ __forceinline__ double iem1t(int sidx, int s, int p) const {
    const bool minus = (sidx == 0) == (s > 0);
    if (ON) return minus ? iem_m : iem_p;
    return __ldg(pair_iem1 + (minus ? 0 : n_pairs) + p);
  }
  template <bool ON> __device__ __forceinline__ int sitet(int sidx, int p) const { return ON ? p : __ldg(pair_site + sidx * n_pairs + p); }
  // pair index of an extended slot, for the E / site accessors (not needed, hence not loaded, in the on-site model)
  __device__ __forceinline__ int pair_of(const int32_t* pairs, int slot) const { return onsite ? 0 : pairs[slot]; }
  // displacement index between the sites two vertices (pairs pi, pj) occupy in spin sector sidx
  __device__ __forceinline__ int pdisp(int sidx, int pi, int pj) const { return disp(site(sidx, pi), site(sidx, pj)); }
  __device__ __forceinline__ int disp(int i, int j) const {
    const int xi = i % Lx, yi = i / Lx, xj = j % Lx, yj = j / Lx;
    int dx = xi - xj; if (dx < 0) dx += Lx;
    int dy = yi - yj; if (dy < 0) dy += Ly;
    return dx + Lx * dy;
  }
  // positive-convention propagator g = -G0 by linear interpolation, antiperiodic in tau
  __device__ __forceinline__ double g(int d, double dtau) const {
    double sg = 1.0;
    if (dtau < 0.0) { sg = -1.0; dtau += beta; }
    const double x = dtau * tau_scale;
    int m = (int)floor(x);
    if (m > M - 1) m = M - 1;
    const double f = x - (double)m;
    const double* T = table + (size_t)d * (M + 1);
    const double t0 = __ldg(T + m), t1 = __ldg(T + m + 1);
    return -sg * (t0 + f * (t1 - t0));
  }
};

__device__ __forceinline__ void l2_prefetch(const void* p) { asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p)); }

// ---------------------------------------------------------------- Philox4x32-10 (device + host)
__host__ __device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                       uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__host__ __device__ __forceinline__ double unif53(uint32_t a, uint32_t b) {
  const uint64_t u = ((uint64_t)a << 21) | (uint64_t)(b >> 11);
  return (double)u * (1.0 / 9007199254740992.0);
}

// 8-byte asynchronous global -> shared copy (LDGSTS) and the wait for all copies this thread has issued: used by the S3
// kernels to gather the next proposal's scattered entries of N behind the current proposal
__device__ __forceinline__ void cp_async_8(void* smem_dst, const void* gsrc) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

}  // namespace ctaux
