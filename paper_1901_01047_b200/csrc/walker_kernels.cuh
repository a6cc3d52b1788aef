// Kernels of the CT-AUX walker hot path other than the GEMM tiles.
//   S1  k_build_A, k_prep_fill     (G0 interpolation, A and candidate rows/columns)
//   S3  k_prep_window, k_propose   (Philox streams, Metropolis over the delayed block)
//   S4  k_build_uv                 (U = X[:,J], V^T = rows J of N_ext)
// Formulas: SURVEY.md Appendix A (derived from Eq. (19)-(27)); DESIGN.md.
#pragma once
#include "walker_state.cuh"

namespace ctaux {

// ---------------------------------------------------------------------------------------------
// reset: walker w draws init_k vertices from Philox(counter=(i,0,0,0), key=seed)
__global__ void k_init_config(DevCtx c, const uint64_t* seeds, int init_k) {
  const int w = blockIdx.x;
  WalkerState& st = c.ws[w];
  const uint32_t k0 = (uint32_t)(seeds[w] & 0xffffffffu), k1 = (uint32_t)(seeds[w] >> 32);
  const size_t off = c.cfg_off(w, 0);
  for (int i = threadIdx.x; i < init_k; i += blockDim.x) {
    uint32_t r[4];
    philox4x32_10((uint32_t)i, 0u, 0u, 0u, k0, k1, r);
    double tau = c.beta * unif53(r[2], r[3]);
    if (tau >= c.beta) tau = nextafter(c.beta, 0.0);
    c.cfg_spin[off + i] = ((r[0] >> 1) & 1u) ? -1 : +1;
    c.cfg_site[off + i] = (int32_t)(((uint64_t)r[1] * (uint64_t)c.n_pairs) >> 32);   // pair index (= site in the on-site model)
    c.cfg_tau[off + i] = tau;
    c.cfg_id[off + i] = (uint64_t)i;
  }
  if (threadIdx.x == 0) {
    WalkerState z;
    memset(&z, 0, sizeof(z));
    z.key0 = k0; z.key1 = k1;
    z.k = init_k; z.k_new = init_k;
    z.next_id = (uint64_t)init_k;
    z.sign = 1;
    z.min_margin = 1e300;
    st = z;
  }
}

// set_state: configuration already copied into buffer 0 by the host; fill in the scalars
__global__ void k_set_state(DevCtx c, const uint64_t* seeds, const int32_t* k, const uint64_t* next_id,
                            const uint64_t* p) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= c.B) return;
  WalkerState z;
  memset(&z, 0, sizeof(z));
  z.key0 = (uint32_t)(seeds[w] & 0xffffffffu); z.key1 = (uint32_t)(seeds[w] >> 32);
  z.k = k[w]; z.k_new = k[w];
  z.next_id = next_id[w]; z.p = p[w];
  z.sign = 1;
  z.min_margin = 1e300;
  c.ws[w] = z;
}

// Batched hand-over of the configurations (ctaux_set_state / ctaux_get_config_all): the host moves ONE packed array
// per field, [B][max_k] (walker w at offset w*max_k), and these kernels scatter it into / gather it from the per-walker
// configuration buffers, converting the auxiliary spins between the int8 of the ABI and the int32 kept on the device.
struct PackedCfg { int32_t* k; uint64_t* id; int32_t* site; double* tau; int8_t* spin; };

// live block of every N_sigma into the host layout of ctaux_get_N_all: matrix (w, spin) at (2w + spin) max_k^2, ld = k_w
__global__ void k_pack_N(DevCtx c, double* out) {
  const int prob = blockIdx.y, w = prob >> 1, sp = prob & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  const double* N = c.N(w, sp, st.n_cur);
  double* dst = out + (size_t)prob * c.max_k * c.max_k;
  for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < k * k; idx += gridDim.x * blockDim.x) {
    const int j = idx / k, i = idx - j * k;
    dst[idx] = N[(size_t)j * c.ld + i];
  }
}

__global__ void k_scatter_state(DevCtx c, PackedCfg pk) {   // -> configuration buffer 0 of every walker
  const int w = blockIdx.y;
  const int k = pk.k[w];
  const size_t off = c.cfg_off(w, 0), src = (size_t)w * c.max_k;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < k; i += gridDim.x * blockDim.x) {
    c.cfg_site[off + i] = pk.site[src + i];
    c.cfg_tau[off + i] = pk.tau[src + i];
    c.cfg_id[off + i] = pk.id[src + i];
    c.cfg_spin[off + i] = (int32_t)pk.spin[src + i];
  }
}

__global__ void k_gather_state(DevCtx c, PackedCfg pk) {    // current configuration buffer of every walker ->
  const int w = blockIdx.y;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  const size_t off = c.cfg_off(w, st.cfg_cur), dst = (size_t)w * c.max_k;
  if (blockIdx.x == 0 && threadIdx.x == 0) pk.k[w] = k;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < k; i += gridDim.x * blockDim.x) {
    pk.site[dst + i] = c.cfg_site[off + i];
    pk.tau[dst + i] = c.cfg_tau[off + i];
    pk.id[dst + i] = c.cfg_id[off + i];
    pk.spin[dst + i] = (int8_t)c.cfg_spin[off + i];
  }
}

// S1: A_sigma[i][j] = delta_ij E_j - g_ij (E_j - 1) into the current N buffer (column-major).
__global__ void k_build_A(DevCtx c, int into_other) {
  const int w = blockIdx.y >> 1, sp = blockIdx.y & 1;
  const WalkerState& st = c.ws[w];
  const int k = st.k;
  const size_t off = c.cfg_off(w, st.cfg_cur);
  double* A = c.N(w, sp, into_other ? (st.n_cur ^ 1) : st.n_cur);
  const size_t total = (size_t)k * k;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(idx % k), j = (int)(idx / k);
    const double Ej = c.E(sp, c.cfg_spin[off + j], c.cfg_site[off + j]);
    double v;
    if (i == j) v = Ej - c.g00 * (Ej - 1.0);
    else v = -c.g(c.pdisp(sp, c.cfg_site[off + i], c.cfg_site[off + j]), c.cfg_tau[off + i] - c.cfg_tau[off + j]) * (Ej - 1.0);
    A[(size_t)j * c.ld + i] = v;
  }
}

// ---------------------------------------------------------------------------------------------
// Start of a ctaux_sweep chunk.
__global__ void k_begin_sweeps(DevCtx c, int n_sweeps, int n_props) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w == 0) { c.n_active[0] = c.B; c.n_active[1] = 0; }
  if (w >= c.B) return;
  c.ws[w].sweeps_left = n_sweeps;
  c.ws[w].props_left = n_props;     // > 0: ctaux_propose (a partial sweep first)
  c.ws[w].active = 1;
  c.ws[w].r = 0;
}

// S3a: expand the next window of proposals of every walker.  Philox is counter based, so the
// words of proposals p, p+1, ... are known before any of them is decided.
// Proposal p: wA = Philox(p_lo, p_hi, 0, 1), wB = Philox(p_lo, p_hi, 1, 1).
__global__ void __launch_bounds__(1024) k_prep_window(DevCtx c) {
  const int w = blockIdx.x;
  WalkerState& st = c.ws[w];
  __shared__ int s_scan[1024];
  __shared__ int s_win;
  const int tid = threadIdx.x;
  if (!st.active || st.status) {
    if (tid == 0) { st.m = 0; st.win = 0; st.r = 0; st.n_src = st.n_cur; atomicMax(c.n_active + 1, st.k); }
    return;
  }
  const int k = st.k;
  const uint64_t p = st.p + (uint64_t)tid;
  uint32_t wa[4] = {0, 0, 0, 0}, wb[4] = {0, 0, 0, 0};
  const bool in = tid < c.winmax;
  if (in) {
    philox4x32_10((uint32_t)(p & 0xffffffffu), (uint32_t)(p >> 32), 0u, 1u, st.key0, st.key1, wa);
    philox4x32_10((uint32_t)(p & 0xffffffffu), (uint32_t)(p >> 32), 1u, 1u, st.key0, st.key1, wb);
  }
  const uint32_t mtype = c.flips ? (uint32_t)(((uint64_t)wb[2] * 3u) >> 32) : (wa[0] & 1u);
  const int is_ins = (in && mtype == 0u) ? 1 : 0;
  // inclusive scan of is_ins over the CTA
  s_scan[tid] = is_ins;
  if (tid == 0) s_win = c.winmax;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {
    int v = 0;
    if (tid >= off) v = s_scan[tid - off];
    __syncthreads();
    s_scan[tid] += v;
    __syncthreads();
  }
  const int cand = s_scan[tid] - is_ins;  // exclusive: index of this insertion among candidates
  // the window ends before the first insertion that has no candidate slot left
  if (is_ins && cand == c.mmax) s_win = tid;  // exactly one thread satisfies this
  __syncthreads();
  const int win = s_win;
  if (in && tid < win) {
    PropInfo pi;
    pi.type_cand = mtype | ((uint32_t)(is_ins ? cand : 0) << 2);
    pi.w1 = wa[1];
    pi.u = unif53(wb[0], wb[1]);
    c.prop[(size_t)w * c.winmax + tid] = pi;
    if (is_ins) {  // candidate vertex -> extended slot k + cand of the current configuration buffer
      const size_t off = c.cfg_off(w, st.cfg_cur) + k + cand;
      double tau = c.beta * unif53(wa[2], wa[3]);
      if (tau >= c.beta) tau = nextafter(c.beta, 0.0);
      c.cfg_spin[off] = ((wa[0] >> 1) & 1u) ? -1 : +1;
      c.cfg_site[off] = (int32_t)(((uint64_t)wa[1] * (uint64_t)c.n_pairs) >> 32);
      c.cfg_tau[off] = tau;
      c.cfg_id[off] = ~0ull;
    }
  }
  if (tid == 0) {
    const int m = (win > 0) ? (s_scan[win - 1]) : 0;
    st.m = m < c.mmax ? m : c.mmax;
    st.win = win;
    st.r = 0;
    st.n_src = st.n_cur;
  }
}

// S1 for the block: candidate rows  Bm[c,j] = g(c,j)(E_j - 1)  (per spin),
// candidate columns gxC[i,c] = g(i,c) over ALL extended slots i (spin independent), and the
// [*, cand] block of N_ext (zeros + identity): a non-interacting slot has column e_c in A,
// hence in N as well.
__global__ void k_prep_fill(DevCtx c) {
  const int w = blockIdx.y;
  const WalkerState& st = c.ws[w];
  const int m = st.m, k = st.k;
  if (m == 0) return;
  const int n = k + m;
  const size_t off = c.cfg_off(w, st.cfg_cur);
  const int32_t* site = c.cfg_site + off;
  const double* tau = c.cfg_tau + off;
  const int32_t* spin = c.cfg_spin + off;
  double* Bm0 = c.Bm + ((size_t)w * 2 + 0) * (size_t)c.ldm * c.cap;
  double* Bm1 = c.Bm + ((size_t)w * 2 + 1) * (size_t)c.ldm * c.cap;
  double* gx0 = c.gxC + ((size_t)w * 2 + 0) * c.ld * c.ldm;
  double* gx1 = c.gxC + ((size_t)w * 2 + 1) * c.ld * c.ldm;
  double* N0 = c.N(w, 0, st.n_cur);
  double* N1 = c.N(w, 1, st.n_cur);
  const size_t total = (size_t)n * m;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(idx % n), cc = (int)(idx / n);
    const int sc = k + cc;
    const int pi = site[i], pc = site[sc];                    // pair indices; the two spin sectors may see different sites
    const int i0 = c.site(0, pi), i1 = c.site(1, pi), c0 = c.site(0, pc), c1 = c.site(1, pc);
    const bool same = (i0 == i1) && (c0 == c1);                // on-site pairs: one interpolation serves both spins
    // column: g(i, c), stored n-contiguous (the "N-major" right operand of gemm_tma.cuh)
    double gic0, gic1;
    if (i == sc) { gic0 = c.g00; gic1 = c.g00; }
    else {
      gic0 = c.g(c.disp(i0, c0), tau[i] - tau[sc]);
      gic1 = same ? gic0 : c.g(c.disp(i1, c1), tau[i] - tau[sc]);
    }
    gx0[(size_t)i * c.ldm + cc] = gic0;
    if (!c.onsite) gx1[(size_t)i * c.ldm + cc] = gic1;   // (on-site model: both sectors read the sp = 0 copy)
    // [*, cand] block of N_ext
    const double e = (i == sc) ? 1.0 : 0.0;
    N0[(size_t)sc * c.ld + i] = e;
    N1[(size_t)sc * c.ld + i] = e;
    // row: g(c, j)(E_j - 1), only against the live vertices j < k
    if (i < k) {
      const double gci0 = c.g(c.disp(c0, i0), tau[sc] - tau[i]);
      const double gci1 = same ? gci0 : c.g(c.disp(c1, i1), tau[sc] - tau[i]);
      Bm0[(size_t)i * c.ldm + cc] = gci0 * (c.E(0, spin[i], pi) - 1.0);
      Bm1[(size_t)i * c.ldm + cc] = gci1 * (c.E(1, spin[i], pi) - 1.0);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// S3: serial Metropolis over the window, one CTA per walker, both spins.
// X_sigma = N_ext - G_ext (n x n, never formed):
//   X[i,j] = (delta_ij - N_ext[i,j]) / (E0_j - 1)      j a block-start vertex
//          =  delta_ij - Gx[i, j-k0]                   j a candidate
// Buffered changes J = (j_1..j_r), dE_a;  S_ab = delta_ab/dE_a + X[j_a, j_b];
// det A_{r+1} / det A_r = dE_new (s_nn - s_row S^-1 s_col)
// Slot the NEXT proposal of the window will meet if the current one (type, slot, list position j) is rejected (ns) or
// accepted (nsA); -1 where it needs no gather (no vertex to pick, or the removal of an in-block insert, which reads
// S^-1 only).  An insert names its candidate slot directly; a removal / flip picks by position in the live list, which
// an accepted insert extends by `slot` and an accepted removal shifts.  Shared by k_propose and k_propose_cl.
struct NextSlots { int type, ns, nsA; };
__device__ __forceinline__ NextSlots next_slots(const PropInfo pn, int k0, int kcur, const int* live, int type, int slot, int j) {
  NextSlots o;
  o.type = (int)(pn.type_cand & 3u);
  o.ns = o.nsA = -1;
  if (o.type == 0) {
    o.ns = o.nsA = k0 + (int)(pn.type_cand >> 2);
  } else {
    if (kcur > 0) o.ns = live[(int)(((uint64_t)pn.w1 * (uint64_t)kcur) >> 32)];
    if (type == 0) {            // accepted insert: the list (length kcur) grows by `slot` at its end
      const int jn = (int)(((uint64_t)pn.w1 * (uint64_t)(kcur + 1)) >> 32);
      o.nsA = jn == kcur ? slot : live[jn];
    } else if (type == 1) {     // accepted removal of position j: later positions shift down
      if (kcur > 1) { const int jn = (int)(((uint64_t)pn.w1 * (uint64_t)(kcur - 1)) >> 32); o.nsA = live[jn + (jn >= j ? 1 : 0)]; }
    } else {
      o.nsA = o.ns;             // accepted flip: same list
    }
    if (o.type == 1 && o.ns >= k0) o.ns = -1;
    if (o.type == 1 && o.nsA >= k0) o.nsA = -1;
  }
  return o;
}
// X[i, j] from the raw entry of N_ext (j < k0: a block-start column, iem_j = 1/(E0_j - 1)) or of G_ext (a candidate column)
__device__ __forceinline__ double x_from_raw(double raw, bool diag, bool blockstart_col, double iem_j) {
  const double d = (diag ? 1.0 : 0.0) - raw;
  return blockstart_col ? d * iem_j : d;
}

constexpr int kPropThreads = 256;
constexpr int kGroup = kPropThreads / 2;  // threads per spin

struct ProposeSmem {
  // byte offsets into dynamic shared memory
  int sinv, scol, srow, tv, tpv, jiem, red, snn, spec, live0, live1, spin, J, jpos, prop, flip, total;
};

__host__ __device__ inline ProposeSmem propose_smem_layout(int cap, int delay, int winmax, bool sinv_smem) {
  ProposeSmem L;
  int o = 0;
  const int lds = delay | 1;
  L.sinv = o; o += sinv_smem ? 2 * lds * delay * 8 : 0;
  L.scol = o; o += 2 * delay * 8;
  L.srow = o; o += 2 * delay * 8;
  L.tv = o; o += 2 * delay * 8;
  L.tpv = o; o += 2 * delay * 8;
  L.jiem = o; o += 2 * delay * 8;
  L.red = o; o += 2 * 2 * 8 * 8;
  L.snn = o; o += 4 * 8;
  L.spec = o; o += 2 * (4 * delay + 2) * 8;   // speculative gather, 2 hypotheses: [2 spins][s_col | s_row][delay] raw entries + 2 diagonals
  L.prop = o; o += winmax * 16;
  L.live0 = o; o += cap * 4;
  L.live1 = o; o += cap * 4;
  L.J = o; o += delay * 4;
  L.jpos = o; o += (winmax + 1) * 4;
  L.spin = o; o += (cap + 15) / 16 * 16;
  L.flip = o; o += (cap + 15) / 16 * 16;
  L.total = o;
  return L;
}

template <bool sinv_smem, bool ONSITE>   // S^-1 of both spins in shared memory (delay <= ~100) or in global memory; model class
__global__ void __launch_bounds__(kPropThreads) k_propose(DevCtx c) {
  extern __shared__ __align__(16) unsigned char smraw[];
  const int w = blockIdx.x, tid = threadIdx.x;
  WalkerState& st = c.ws[w];
  if (!st.active || st.status || st.win == 0) return;
  const ProposeSmem L = propose_smem_layout(c.cap, c.delay, c.winmax, sinv_smem);
  const int sp = tid / kGroup, lt = tid % kGroup;
  const int lds = sinv_smem ? (c.delay | 1) : c.ldr;
  double* Sbase = sinv_smem ? reinterpret_cast<double*>(smraw + L.sinv)
                            : (c.Sinv + (size_t)w * 2 * (size_t)c.ldr * c.delay);
  const size_t sstride = (size_t)lds * c.delay;  // spin stride of S^-1
  double* Sv = Sbase + (size_t)sp * sstride;
  double* scol = reinterpret_cast<double*>(smraw + L.scol) + sp * c.delay;
  double* srow = reinterpret_cast<double*>(smraw + L.srow) + sp * c.delay;
  double* tv = reinterpret_cast<double*>(smraw + L.tv) + sp * c.delay;
  double* tpv = reinterpret_cast<double*>(smraw + L.tpv) + sp * c.delay;
  double* jiem = reinterpret_cast<double*>(smraw + L.jiem) + sp * c.delay;   // 1/(E0 - 1) of the buffered block-start vertices
  double* red = reinterpret_cast<double*>(smraw + L.red);   // [2][8] dot products, [2][8] sums of magnitudes
  double* snn2 = reinterpret_cast<double*>(smraw + L.snn);  // [2 parities][2 spins]
  PropInfo* prop = reinterpret_cast<PropInfo*>(smraw + L.prop);
  int* live = reinterpret_cast<int*>(smraw + L.live0);
  int* live_alt = reinterpret_cast<int*>(smraw + L.live1);
  int* Js = reinterpret_cast<int*>(smraw + L.J);
  int* jpos = reinterpret_cast<int*>(smraw + L.jpos);  // candidate index -> position in J (-1: not buffered)
  signed char* spin_s = reinterpret_cast<signed char*>(smraw + L.spin);
  signed char* flipped = reinterpret_cast<signed char*>(smraw + L.flip);   // 1: block-start vertex flipped in this block

  const int k0 = st.k, m = st.m, win = st.win, n = k0 + m;
  const int cfg_old = st.cfg_cur;
  const size_t off_old = c.cfg_off(w, cfg_old), off_new = c.cfg_off(w, cfg_old ^ 1);
  const double* Ncur = c.N(w, sp, st.n_cur);
  const double* Gx = c.Gx + ((size_t)w * 2 + sp) * (size_t)c.ld * c.mmax;
  const int ld = c.ld;
  const int32_t* pair_g = c.cfg_site + off_old;   // pair index of every extended slot

  for (int i = tid; i < n; i += kPropThreads) spin_s[i] = (signed char)c.cfg_spin[off_old + i];
  for (int i = tid; i < k0; i += kPropThreads) { live[i] = i; flipped[i] = 0; }
  for (int i = tid; i < win; i += kPropThreads) prop[i] = c.prop[(size_t)w * c.winmax + i];
  for (int i = tid; i <= c.winmax; i += kPropThreads) jpos[i] = -1;
  __syncthreads();

  // X[i, j] with the factor 1/(E0_j - 1) of a block-start column j handed in by the caller
  auto X = [&](int i, int j, double iem_j) -> double {
    const double dlt = (i == j) ? 1.0 : 0.0;
    if (j < k0) return (dlt - Ncur[(size_t)j * ld + i]) * iem_j;
    return dlt - Gx[(size_t)(j - k0) * ld + i];
  };

  int kcur = k0, r = 0, len = k0;
  int props_left = st.props_left, sweeps_left = st.sweeps_left;
  uint64_t next_id = st.next_id, p = st.p;
  int sign = st.sign, status = 0, consumed = 0;
  int64_t acc_ins = 0, acc_rem = 0, acc_flip = 0, sweeps_done = 0;
  double mm_du = st.min_margin, mm_aR = 1.0, sum_k = 0.0;   // decision margin as a fraction (no division per proposal)
  int64_t log_count = st.log_count;
  bool finished = false;
  int guard_end = 0;
  double errlvl = 1.0;  // rounding-error level of S^-1 in units of eps (largest amplification accepted so far)
  // Speculative gather: the entries X(J[a], slot), X(slot, J[a]) and the diagonal entry of the NEXT proposal are loaded
  // while the current one is evaluated (a third of a proposal's latency is this dependent gather from L2 / HBM).  The
  // loads assume the current proposal is rejected, plus one entry for J[r] = the current slot in case it is accepted;
  // they are used when the next proposal really meets that slot and that J (checked below), else gathered again.
  // The loads are asynchronous copies into shared memory (LDGSTS): register loads kept in flight across a proposal
  // tie up the warp's scoreboards and were measured SLOWER than no speculation at all.
  // Buffer 0 holds the entries for the slot the next proposal meets if the current one is REJECTED, buffer 1 those for
  // the slot it meets if the current one is ACCEPTED, when that is a different slot (a removal or flip picks its target
  // by position in the live list, which an accepted move shifts); where the two slots agree buffer 0 serves both.
  const int spec_stride = 4 * c.delay + 2;
  double* spec_own = reinterpret_cast<double*>(smraw + L.spec) + (sp * 2 + (lt >> 6)) * c.delay;   // this thread's role
  double* spec_dg = reinterpret_cast<double*>(smraw + L.spec) + 4 * c.delay + sp;
  int spec_slot = -1, specA_slot = -1, specA_buf = 0, spec_r = -1, spec_jver = -1, spec_type = -1, jver = 0;

  for (int i = 0; i < win; ++i) {
    if (props_left == 0) {
      if (sweeps_left == 0) { finished = true; break; }
      --sweeps_left;
      props_left = kcur > 16 ? kcur : 16;
    }
    const PropInfo pi = prop[i];
    const int type = (int)(pi.type_cand & 3u);
    int slot = -1, j = -1;
    double pref = 0.0;
    if (type == 0) {
      slot = k0 + (int)(pi.type_cand >> 2);
      pref = c.K / (double)(kcur + 1);
    } else if (kcur > 0) {
      j = (int)(((uint64_t)pi.w1 * (uint64_t)kcur) >> 32);
      slot = live[j];
      pref = type == 1 ? (double)kcur / c.K : 1.0;
      // A vertex already changed in this block (flipped, or inserted and now to be flipped) is not touched a
      // second time inside the block: the block is flushed BEFORE this proposal, which then meets an untouched
      // vertex (exact; the insert-then-remove pair keeps its own in-block treatment below).
      if ((type == 2 && (slot >= k0 || flipped[slot])) || (type == 1 && slot < k0 && flipped[slot])) { guard_end = 2; break; }
    }
    bool accept = false;
    double R = 0.0, stil_own = 1.0, iem_own = 0.0;
    double amp_n0 = 1.0, amp_n1 = 1.0, amp_d0 = 1.0, amp_d1 = 1.0;   // amp = max(n0/d0, n1/d1), divided on accept only
    // removal of a vertex inserted earlier in this block: the two changes of that slot cancel, so
    // the buffered insertion is taken OUT of the block (exact treatment of a twice-touched spin,
    // PAPER.md:228): ratio = (S^-1)_aa / dE_a, then S^-1 is downdated.
    const bool down = (type == 1 && slot >= k0);
    int apos = -1;
    if (down) {
      apos = jpos[slot - k0];
      const int s = spin_s[slot];
      const double sa0 = Sbase[apos + (size_t)apos * lds], sa1 = Sbase[sstride + apos + (size_t)apos * lds];
      const int pr = (ONSITE ? 0 : pair_g[slot]);
      R = pref * ((sa0 / (c.template Et<ONSITE>(0, s, pr) - 1.0)) * (sa1 / (c.template Et<ONSITE>(1, s, pr) - 1.0)));
      accept = pi.u < fabs(R);
      stil_own = sp == 0 ? sa0 : sa1;
    } else if (slot >= 0) {
      const int s = spin_s[slot];
      const int pr = (ONSITE ? 0 : pair_g[slot]);
      const double E0 = c.template Et<ONSITE>(0, s, pr), E1 = c.template Et<ONSITE>(1, s, pr);
      // column change of A: insert 1 -> E, remove E -> 1, flip E(s) -> E(-s)
      const double dE0 = (type == 0) ? (E0 - 1.0) : (type == 1 ? (1.0 - E0) : (c.template Et<ONSITE>(0, -s, pr) - E0));
      const double dE1 = (type == 0) ? (E1 - 1.0) : (type == 1 ? (1.0 - E1) : (c.template Et<ONSITE>(1, -s, pr) - E1));
      const double dE_own = sp == 0 ? dE0 : dE1;
      const double iem_slot = c.template iem1t<ONSITE>(sp, s, pr);     // 1/(E0 - 1) of this slot's column (used when slot < k0)
      iem_own = iem_slot;
      // thread roles inside a spin group of 128: half 0 builds s_col and t = S^-1 s_col (and the dot
      // product), half 1 builds s_row and t' = s_row^T S^-1; 64 rows per pass
      const int half = lt >> 6, la = lt & 63;
      double* snn = snn2 + (i & 1) * 2;   // double buffered: read after the second barrier of this proposal
      const bool hitR = spec_slot == slot && spec_r == r, hitA = specA_slot == slot && spec_r + 1 == r;
      const bool hit = spec_type == type && spec_jver == jver && (hitR || hitA);
      const int hbuf = (hitR ? 0 : specA_buf) * spec_stride;
      cp_async_wait_all();     // this thread's own copies of the previous proposal (long done; it reads only those)
      if (hit) {
        for (int a = la; a < r; a += 64) {
          const int ja = Js[a];
          const double raw = spec_own[hbuf + a];
          if (half == 0) scol[a] = x_from_raw(raw, ja == slot, slot < k0, iem_slot);      // X(ja, slot)
          else srow[a] = x_from_raw(raw, ja == slot, ja < k0, jiem[a]);                  // X(slot, ja)
        }
        if (lt == 0) {
          const double raw = spec_dg[hbuf];
          if (slot < k0 && type == 1) snn[sp] = -raw * iem_slot;
          else snn[sp] = 1.0 / dE_own + x_from_raw(raw, true, slot < k0, iem_slot);
        }
      } else {
        for (int a = la; a < r; a += 64) {
          const int ja = Js[a];
          if (half == 0) scol[a] = X(ja, slot, iem_slot);
          else srow[a] = X(slot, ja, jiem[a]);
        }
        if (lt == 0) {
          // diagonal entry 1/dE + X[slot,slot]; for a block-start vertex (removal, dE = 1 - E) this is
          // -N[slot,slot]/(E-1) exactly, written so that nothing cancels
          if (slot < k0 && type == 1) snn[sp] = -Ncur[(size_t)slot * ld + slot] * iem_slot;
          else snn[sp] = 1.0 / dE_own + X(slot, slot, iem_slot);
        }
      }
      // issue the copies of the next proposal (consumed one iteration later: their latency hides behind this proposal)
      spec_slot = -1; specA_slot = -1; specA_buf = 0;
      if (i + 1 < win) {
        const NextSlots nx = next_slots(prop[i + 1], k0, kcur, live, type, slot, j);
        const int tn = nx.type, ns = nx.ns, nsA = nx.nsA;
        spec_type = tn; spec_r = r; spec_jver = jver;
        auto issue = [&](int nsl, int buf) {
          const double* coln = nsl < k0 ? Ncur + (size_t)nsl * ld : Gx + (size_t)(nsl - k0) * ld;    // column of N_ext / G_ext
          for (int a = la; a <= r; a += 64) {
            const int ja = a < r ? Js[a] : slot;
            const double* src = half == 0 ? coln + ja
                                          : (ja < k0 ? Ncur + (size_t)ja * ld + nsl : Gx + (size_t)(ja - k0) * ld + nsl);
            cp_async_8(spec_own + buf * spec_stride + a, src);
          }
          if (lt == 0) cp_async_8(spec_dg + buf * spec_stride, coln + nsl);
        };
        if (ns >= 0) { spec_slot = ns; issue(ns, 0); }
        if (nsA >= 0) {
          specA_slot = nsA;
          if (nsA != ns) { specA_buf = 1; issue(nsA, 1); }
        }
      }
      __syncthreads();
      double part = 0.0, apart = 0.0;
      for (int a = la; a < r; a += 64) {
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
        int b = 0;
        if (half == 0) {
          const double* Sa = Sv + a;
          for (; b + 3 < r; b += 4) {
            s0 += Sa[(size_t)b * lds] * scol[b];
            s1 += Sa[(size_t)(b + 1) * lds] * scol[b + 1];
            s2 += Sa[(size_t)(b + 2) * lds] * scol[b + 2];
            s3 += Sa[(size_t)(b + 3) * lds] * scol[b + 3];
          }
          for (; b < r; ++b) s0 += Sa[(size_t)b * lds] * scol[b];
          const double t = (s0 + s1) + (s2 + s3);
          tv[a] = t;
          part += srow[a] * t;
          apart += fabs(srow[a] * t);
        } else {
          const double* Sa = Sv + (size_t)a * lds;
          for (; b + 3 < r; b += 4) {
            s0 += srow[b] * Sa[b];
            s1 += srow[b + 1] * Sa[b + 1];
            s2 += srow[b + 2] * Sa[b + 2];
            s3 += srow[b + 3] * Sa[b + 3];
          }
          for (; b < r; ++b) s0 += srow[b] * Sa[b];
          tpv[a] = (s0 + s1) + (s2 + s3);
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        part += __shfl_xor_sync(0xffffffffu, part, o);
        apart += __shfl_xor_sync(0xffffffffu, apart, o);
      }
      if ((tid & 31) == 0) { red[sp * 8 + (lt >> 5)] = part; red[16 + sp * 8 + (lt >> 5)] = apart; }
      __syncthreads();
      const double dot0 = (red[0] + red[1]) + (red[2] + red[3]);
      const double dot1 = (red[8] + red[9]) + (red[10] + red[11]);
      const double stil0 = snn[0] - dot0, stil1 = snn[1] - dot1;
      // Numerical guard (ctaux_params.guard_amp): the bordered evaluation s_nn - s_row S^-1 s_col
      // amplifies rounding errors by amp = (|s_nn| + sum |s_row_a t_a|) / |result|, on top of the error
      // level S^-1 already carries.  When that product exceeds the guard the block is flushed BEFORE
      // this proposal, which is then evaluated first thing in the next block straight from the
      // updated N (r = 0: no bordering).  Chain-neutral: only where blocks end.
      {
        const double ad0 = (red[16] + red[17]) + (red[18] + red[19]);
        const double ad1 = (red[24] + red[25]) + (red[26] + red[27]);
        // amp_s * errlvl > guard  <=>  num_s * errlvl > guard * den_s: no division on the decision path (amp itself is
        // only needed when the proposal is accepted)
        const double num0 = fabs(snn[0]) + ad0, num1 = fabs(snn[1]) + ad1;
        const double den0 = fmax(fabs(stil0), 1e-300), den1 = fmax(fabs(stil1), 1e-300);
        if (r > 0 && (num0 * errlvl > c.guard_amp * den0 || num1 * errlvl > c.guard_amp * den1)) { guard_end = 1; break; }
        amp_n0 = num0; amp_n1 = num1; amp_d0 = den0; amp_d1 = den1;
      }
      stil_own = sp == 0 ? stil0 : stil1;
      R = pref * ((dE0 * stil0) * (dE1 * stil1));
      accept = pi.u < fabs(R);
    }
    if (tid == 0) {
      if (log_count < (int64_t)c.log_capacity) {
        LogEntry e;
        e.p = p; e.type = type;
        e.arg = (type == 0) ? c.cfg_site[off_old + slot] : j;
        e.tau = (type == 0) ? c.cfg_tau[off_old + slot] : 0.0;
        e.spin = (type == 0) ? (int)spin_s[slot] : 0;
        e.accepted = accept ? 1 : 0;
        e.R = R; e.u = pi.u;
        c.log[(size_t)w * c.log_capacity + log_count] = e;
      }
    }
    ++log_count;
    if (slot >= 0) {
      const double aR = fmax(fabs(R), 1e-300), du = fabs(pi.u - fabs(R));
      if (du * mm_aR < mm_du * aR) { mm_du = du; mm_aR = aR; }      // smallest du / aR, divided once at write-back
    }
    sum_k += (double)kcur;
    if (accept && type == 0 && kcur + 1 > c.max_k) { status = -2; break; }  // CTAUX_ECAPACITY
    if (accept && down) {
      // S^-1 <- S^-1 - S^-1[:,a] S^-1[a,:] / S^-1[a,a], then entry a is replaced by the last one
      const double inv = 1.0 / stil_own;
      for (int a = lt; a < r; a += kGroup) {
        tv[a] = Sv[a + (size_t)apos * lds];
        tpv[a] = Sv[apos + (size_t)a * lds];
      }
      __syncthreads();
      for (int a = lt & 63; a < r; a += 64) {
        const double ta = tv[a] * inv;
        double* Sa = Sv + a;
        for (int b = lt >> 6; b < r; b += 2) Sa[(size_t)b * lds] -= ta * tpv[b];
      }
      __syncthreads();
      const int last = r - 1;
      if (apos != last) {
        for (int b = lt; b < r; b += kGroup) Sv[apos + (size_t)b * lds] = Sv[last + (size_t)b * lds];
        __syncthreads();
        for (int a = lt; a < last; a += kGroup) Sv[a + (size_t)apos * lds] = Sv[a + (size_t)last * lds];
      }
      if (lt == 0 && apos != last) jiem[apos] = jiem[last];
      if (tid == 0) {
        jpos[slot - k0] = -1;
        if (apos != last) {
          const int moved = Js[last];
          Js[apos] = moved;
          if (moved >= k0) jpos[moved - k0] = apos;
        }
      }
      for (int idx = tid; idx < len - 1; idx += kPropThreads) live_alt[idx] = live[idx + (idx >= j ? 1 : 0)];
      int* t = live; live = live_alt; live_alt = t;
      --len; --kcur; ++acc_rem;
      if (R < 0.0) sign = -sign;
      --r; ++jver;      // J was re-ordered: speculative loads of the next proposal are void
    } else if (accept) {
      const double inv = 1.0 / stil_own;
      for (int a = lt & 63; a < r; a += 64) {   // 64 rows x 2 column phases: no integer division
        const double ta = tv[a] * inv;
        double* Sa = Sv + a;
        for (int b = lt >> 6; b < r; b += 2) Sa[(size_t)b * lds] += ta * tpv[b];
      }
      for (int a = lt; a < r; a += kGroup) {
        Sv[a + (size_t)r * lds] = -tv[a] * inv;
        Sv[r + (size_t)a * lds] = -tpv[a] * inv;
      }
      if (lt == 0) { Sv[r + (size_t)r * lds] = inv; jiem[r] = iem_own; }
      if (tid == 0) Js[r] = slot;
      errlvl = fmax(errlvl, amp_n0 * amp_d1 > amp_n1 * amp_d0 ? amp_n0 / amp_d0 : amp_n1 / amp_d1);   // max of the two ratios, one division
      if (type == 0) {
        if (tid == 0) { live[len] = slot; c.cfg_id[off_old + slot] = next_id; jpos[slot - k0] = r; }
        ++len; ++kcur; ++next_id; ++acc_ins;
      } else if (type == 2) {
        if (tid == 0) flipped[slot] = 1;     // the vertex stays in the list; its spin changes at write-back
        ++acc_flip;
      } else {
        for (int idx = tid; idx < len - 1; idx += kPropThreads) live_alt[idx] = live[idx + (idx >= j ? 1 : 0)];
        int* t = live; live = live_alt; live_alt = t;
        --len; --kcur; ++acc_rem;
      }
      if (R < 0.0) sign = -sign;
      ++r;
    }
    if (accept) __syncthreads();   // S^-1, J, the live list changed; a rejected proposal wrote nothing shared
    --props_left; ++consumed; ++p;
    if (props_left == 0) ++sweeps_done;
    if (r == c.delay) break;
  }
  __syncthreads();
  if (props_left == 0 && sweeps_left == 0) finished = true;

  // ---- write back: new list (compacted), S^-1, J, scalars
  int* rowmap = c.rowmap + (size_t)w * c.cap;
  for (int i = tid; i < kcur; i += kPropThreads) {
    const int sl = live[i];
    rowmap[i] = sl;
    c.cfg_site[off_new + i] = c.cfg_site[off_old + sl];
    c.cfg_tau[off_new + i] = c.cfg_tau[off_old + sl];
    c.cfg_spin[off_new + i] = (sl < k0 && flipped[sl]) ? -c.cfg_spin[off_old + sl] : c.cfg_spin[off_old + sl];
    c.cfg_id[off_new + i] = c.cfg_id[off_old + sl];
  }
  if (sinv_smem) {
    double* Sg = c.Sinv + ((size_t)w * 2 + sp) * (size_t)c.ldr * c.delay;
    for (int idx = lt; idx < r * r; idx += kGroup) {
      const int a = idx % r, b = idx / r;
      Sg[a + (size_t)b * c.ldr] = Sv[a + (size_t)b * lds];
    }
  }
  for (int a = tid; a < r; a += kPropThreads) c.J[(size_t)w * c.delay + a] = Js[a];
  if (tid == 0) {
    st.k_new = kcur;
    st.k = kcur;
    st.m = k0;  // block-start order, read by k_build_uv (m is re-set by the next k_prep_window)
    st.cfg_cur = cfg_old ^ 1;
    st.r = r;
    st.n_src = st.n_cur;
    if (r > 0) st.n_cur ^= 1;
    st.next_id = next_id; st.p = p; st.sign = sign;
    st.sweeps_left = sweeps_left; st.props_left = props_left;
    st.acc_ins += acc_ins; st.acc_rem += acc_rem; st.acc_flip += acc_flip; st.sweeps += sweeps_done;
    st.blocks += 1;
    st.guard_ends += guard_end != 0;
    if (r > 0) { st.flushes += 1; st.sum_rank += r; }
    st.log_count = log_count;
    st.min_margin = mm_du / mm_aR; st.sum_k += sum_k;
    st.flops_cand += 2.0 * (2.0 * m * (double)k0 * k0 + 2.0 * (double)n * n * m);
      st.flops_cand_alg += 2.0 * (2.0 * m * (double)k0 * k0 + 2.0 * (double)n * n * (double)acc_ins);   // columns of accepted inserts only
    st.flops_flush += 2.0 * (2.0 * (double)kcur * kcur * r);
    st.flops_usinv += 2.0 * (2.0 * (double)kcur * r * r);
    if (status) st.status = status;
    atomicMax(c.n_active + 1, kcur);   // largest live order, mirrored to the host at every poll (grid sizing)
    if (finished || status) {
      st.active = 0;
      atomicSub(c.n_active, 1);
    }
  }
}

// S4a: U[i', a] = X[rowmap[i'], J[a]],  V[j', a] = N_ext[J[a], rowmap[j']]   (live rows/cols only)
__global__ void k_build_uv(DevCtx c) {
  const int w = blockIdx.y >> 1, sp = blockIdx.y & 1;
  const WalkerState& st = c.ws[w];
  const int r = st.r;
  if (r == 0) return;
  const int kn = st.k_new, k0 = st.m;  // m holds the block-start order after k_propose
  const size_t off_old = c.cfg_off(w, st.cfg_cur ^ 1);
  const double* Nsrc = c.N(w, sp, st.n_src);
  const double* Gx = c.Gx + ((size_t)w * 2 + sp) * (size_t)c.ld * c.mmax;
  double* U = c.Um + ((size_t)w * 2 + sp) * (size_t)c.ld * c.delay;
  double* Vt = c.Vt + ((size_t)w * 2 + sp) * (size_t)c.ldr * c.ld;
  const int* rowmap = c.rowmap + (size_t)w * c.cap;
  const int* J = c.J + (size_t)w * c.delay;
  const int ld = c.ld;
  const size_t total = (size_t)kn * r;
  for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (size_t)gridDim.x * blockDim.x) {
    {  // U: consecutive threads walk down a column of N_ext / Gx
      const int ip = (int)(idx % kn), a = (int)(idx / kn);
      const int i = rowmap[ip], j = J[a];
      const double dlt = (i == j) ? 1.0 : 0.0;
      double x;
      if (j < k0) {
        x = (dlt - Nsrc[(size_t)j * ld + i]) * c.iem1(sp, c.cfg_spin[off_old + j], c.cfg_site[off_old + j]);
      } else {
        x = dlt - Gx[(size_t)(j - k0) * ld + i];
      }
      U[(size_t)a * ld + ip] = x;
    }
    {  // V stored n-contiguous ("N-major" right operand of the flush): V[j', a] = N_ext[J[a], rowmap[j']]
      const int jp = (int)(idx % kn), a = (int)(idx / kn);
      Vt[(size_t)a * ld + jp] = Nsrc[(size_t)rowmap[jp] * ld + J[a]];
    }
  }
}

__global__ void k_set_sign_from_det(DevCtx c, const int* detsign) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= c.B) return;
  c.ws[w].sign = detsign[2 * w] * detsign[2 * w + 1];
}

__global__ void k_count_rebuild(DevCtx c) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= c.B) return;
  WalkerState& st = c.ws[w];
  st.rebuilds += 1;
  st.flops_rebuild += 2.0 * 2.0 * (double)st.k * st.k * st.k;
}

__global__ void k_debug_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint32_t r[4];
  philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1], r);
  out[4 * i] = r[0]; out[4 * i + 1] = r[1]; out[4 * i + 2] = r[2]; out[4 * i + 3] = r[3];
}

}  // namespace ctaux
