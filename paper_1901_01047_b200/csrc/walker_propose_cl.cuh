// S3 for large delays (delay > ~100: S^-1 of both spins no longer fits one SM's shared memory):
// the same serial Metropolis chain as k_propose (walker_kernels.cuh), run by a thread-block CLUSTER of
// two CTAs per walker, one per spin.  Each CTA keeps the S^-1 of its own spin (132 KB at delay 128) in
// its own shared memory (or in L2 when even that does not fit: delay 256), evaluates its spin's
// determinant ratio with 512 threads (4 lanes per row of S^-1), and the two CTAs exchange their
// per-proposal scalars through distributed shared memory: each sends its two values straight into the peer's shared
// memory with st.async, which completes a transaction on the PEER's mbarrier -- data and signal travel together, so no
// cluster barrier (whose release fence waited for every store and look-ahead copy in flight: 40 % of the warp-state
// samples, profiles/r2_propose.md) sits on the per-proposal path.  All
// bookkeeping (live list, J, counters) is replicated, so both CTAs take identical decisions.
// PAPER.md:226-228 (submatrix updates), BASELINE.json config 5 (delay 128 and 256).
#pragma once
#include <cooperative_groups.h>

#include "gemm_tma.cuh"      // mbarrier and distributed-shared-memory helpers
#include "walker_kernels.cuh"

namespace ctaux {

constexpr int kClThreads = 512;

struct ProposeClSmem {
  int sinv, scol, srow, tv, tpv, jiem, red, snn, xch, spec, live0, live1, spin, J, jpos, prop, flip, total;
};
__host__ __device__ inline ProposeClSmem propose_cl_smem_layout(int cap, int delay, int winmax, bool sinv_smem) {
  ProposeClSmem L;
  int o = 0;
  const int lds = delay | 1;
  const int dv = (delay + 1) & ~1;        // the vectors start on 16-byte boundaries (16-byte loads in the two products)
  L.sinv = o; o += sinv_smem ? ((lds * delay * 8 + 15) & ~15) : 0;
  L.scol = o; o += dv * 8;
  L.srow = o; o += dv * 8;
  L.tv = o; o += dv * 8;
  L.tpv = o; o += dv * 8;
  L.jiem = o; o += dv * 8;
  L.red = o; o += 2 * 16 * 8;
  L.snn = o; o += 2 * 8;
  o = (o + 15) & ~15;                 // st.async.v2.f64 wants 16-byte aligned slots
  L.xch = o; o += 2 * 2 * 4 * 8;      // [parity][spin][stil, ampnum, -, -]
  L.spec = o; o += 2 * (2 * delay + 2) * 8;   // speculative gather of the next proposal, 2 hypotheses: [s_col | s_row][delay] raw entries, diagonal
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

template <bool sinv_smem, bool ONSITE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kClThreads, 1) k_propose_cl(DevCtx c) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  extern __shared__ __align__(16) unsigned char smcl[];
  const int w = blockIdx.x >> 1, sp = (int)cluster.block_rank(), tid = threadIdx.x;
  WalkerState& st = c.ws[w];
  if (!st.active || st.status || st.win == 0) return;   // identical in both CTAs of the cluster
  const ProposeClSmem L = propose_cl_smem_layout(c.cap, c.delay, c.winmax, sinv_smem);
  const int lds = sinv_smem ? (c.delay | 1) : c.ldr;
  double* Sv = sinv_smem ? reinterpret_cast<double*>(smcl + L.sinv)
                         : (c.Sinv + ((size_t)w * 2 + sp) * (size_t)c.ldr * c.delay);
  double* scol = reinterpret_cast<double*>(smcl + L.scol);
  double* srow = reinterpret_cast<double*>(smcl + L.srow);
  double* tv = reinterpret_cast<double*>(smcl + L.tv);
  double* tpv = reinterpret_cast<double*>(smcl + L.tpv);
  double* jiem = reinterpret_cast<double*>(smcl + L.jiem);   // 1/(E0 - 1) of the buffered block-start vertices (own spin)
  double* red = reinterpret_cast<double*>(smcl + L.red);    // [16] dot, [16] sum of magnitudes
  double* snn2 = reinterpret_cast<double*>(smcl + L.snn);   // [2 parities]
  double* xch = reinterpret_cast<double*>(smcl + L.xch);
  __shared__ uint64_t xbar[2];      // one mbarrier per slot parity: bytes of exchange e + 1 never count on the phase of exchange e
  const uint32_t xch_peer_addr = mapa_u32(smem_u32(xch), (uint32_t)(sp ^ 1));      // shared::cluster addresses in the peer CTA
  const uint32_t xbar_peer_addr = mapa_u32(smem_u32(xbar), (uint32_t)(sp ^ 1));
  if (tid == 0) { mbar_init(xbar, 1); mbar_init(xbar + 1, 1); mbar_fence_init(); }      // visible to the peer after the first cluster.sync() below
  PropInfo* prop = reinterpret_cast<PropInfo*>(smcl + L.prop);
  int* live = reinterpret_cast<int*>(smcl + L.live0);
  int* live_alt = reinterpret_cast<int*>(smcl + L.live1);
  int* Js = reinterpret_cast<int*>(smcl + L.J);
  int* jpos = reinterpret_cast<int*>(smcl + L.jpos);
  signed char* spin_s = reinterpret_cast<signed char*>(smcl + L.spin);
  signed char* flipped = reinterpret_cast<signed char*>(smcl + L.flip);   // 1: block-start vertex flipped in this block

  const int k0 = st.k, m = st.m, win = st.win, n = k0 + m;
  const int cfg_old = st.cfg_cur;
  const size_t off_old = c.cfg_off(w, cfg_old), off_new = c.cfg_off(w, cfg_old ^ 1);
  const double* Ncur = c.N(w, sp, st.n_cur);
  const double* Gx = c.Gx + ((size_t)w * 2 + sp) * (size_t)c.ld * c.mmax;
  const int ld = c.ld;
  const int32_t* pair_g = c.cfg_site + off_old;   // pair index of every extended slot
  // everything read from the walker state BEFORE the first cluster barrier; rank 0 alone writes it at the end
  int kcur = k0, r = 0, len = k0;
  int props_left = st.props_left, sweeps_left = st.sweeps_left;
  uint64_t next_id = st.next_id, p = st.p;
  int sign = st.sign, status = 0;
  int64_t acc_ins = 0, acc_rem = 0, acc_flip = 0, sweeps_done = 0;
  double mm_du = st.min_margin, mm_aR = 1.0, sum_k = 0.0;   // decision margin as a fraction (no division per proposal)
  int64_t log_count = st.log_count;
  const int n_cur0 = st.n_cur;
  bool finished = false;
  int guard_end = 0;
  double errlvl = 1.0;

  for (int i = tid; i < n; i += kClThreads) spin_s[i] = (signed char)c.cfg_spin[off_old + i];
  for (int i = tid; i < k0; i += kClThreads) { live[i] = i; flipped[i] = 0; }
  for (int i = tid; i < win; i += kClThreads) prop[i] = c.prop[(size_t)w * c.winmax + i];
  for (int i = tid; i <= c.winmax; i += kClThreads) jpos[i] = -1;
  cluster.sync();

  auto X = [&](int i, int j, double iem_j) -> double {   // iem_j = 1/(E0_j - 1) of a block-start column j
    const double dlt = (i == j) ? 1.0 : 0.0;
    if (j < k0) return (dlt - Ncur[(size_t)j * ld + i]) * iem_j;
    return dlt - Gx[(size_t)(j - k0) * ld + i];
  };
  // publish this spin's two scalars to both CTAs, one cluster barrier, read both spins' values
  // Every thread of a CTA holds its own spin's two values already (all threads evaluate the same reduction); thread 0
  // sends them to slot [parity][sp] of the peer and arms the own mbarrier for the 16 bytes the peer sends; everybody
  // waits on the own mbarrier and reads the peer's values.  Slot reuse (two exchanges later) is safe: the peer sends
  // exchange e + 2 only after it has received e + 1, which this CTA's thread 0 sent after a __syncthreads() that all of
  // its threads reach after their reads of slot e.
  int xpar = 0;
  uint32_t xphase = 0;
  auto exchange = [&](double v0, double v1, double (&o0)[2], double (&o1)[2]) {
    if (tid == 0) {
      mbar_expect_tx(xbar + xpar, 16);
      st_async_2f64(xch_peer_addr + (uint32_t)((xpar * 2 + sp) * 4 * 8), v0, v1, xbar_peer_addr + (uint32_t)(xpar * 8));
    }
    mbar_wait(xbar + xpar, xphase);
    const double* theirs = xch + (xpar * 2 + (sp ^ 1)) * 4;
    const double p0 = theirs[0], p1 = theirs[1];
    if (sp == 0) { o0[0] = v0; o0[1] = v1; o1[0] = p0; o1[1] = p1; }
    else { o0[0] = p0; o0[1] = p1; o1[0] = v0; o1[1] = v1; }
    xphase ^= (uint32_t)xpar;      // each barrier is used every other exchange
    xpar ^= 1;
  };

  const int role = tid >> 8, rl = tid & 255;   // role 0: s_col and t; role 1: s_row and t'
  const int row4 = rl >> 2, q4 = rl & 3;       // 64 rows per pass, 4 lanes per row
  const unsigned quad_mask = 0xFu << (tid & 28);   // the 4 lanes of a row leave the row loop together

  // speculative gather of the next proposal's entries (see k_propose): one entry per thread here (delay <= 256 lanes)
  double* spec_own = reinterpret_cast<double*>(smcl + L.spec) + (tid >> 8) * c.delay;
  double* spec_dg = reinterpret_cast<double*>(smcl + L.spec) + 2 * c.delay;
  const int spec_stride = 2 * c.delay + 2;       // buffer 0: next slot if this proposal is rejected, buffer 1: if accepted
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
    const bool down = (type == 1 && slot >= k0);
    int apos = -1;
    if (down) {
      // removal of a vertex inserted earlier in this block: the buffered insertion is taken out
      apos = jpos[slot - k0];
      const int s = spin_s[slot];
      const double sa_own = Sv[apos + (size_t)apos * lds];
      double o0[2], o1[2];
      exchange(sa_own, 0.0, o0, o1);
      const int pr = (ONSITE ? 0 : pair_g[slot]);
      R = pref * ((o0[0] / (c.template Et<ONSITE>(0, s, pr) - 1.0)) * (o1[0] / (c.template Et<ONSITE>(1, s, pr) - 1.0)));
      accept = pi.u < fabs(R);
      stil_own = sa_own;
    } else if (slot >= 0) {
      const int s = spin_s[slot];
      const int pr = (ONSITE ? 0 : pair_g[slot]);
      const double E0 = c.template Et<ONSITE>(0, s, pr), E1 = c.template Et<ONSITE>(1, s, pr);
      // column change of A: insert 1 -> E, remove E -> 1, flip E(s) -> E(-s)
      const double dE0 = (type == 0) ? (E0 - 1.0) : (type == 1 ? (1.0 - E0) : (c.template Et<ONSITE>(0, -s, pr) - E0));
      const double dE1 = (type == 0) ? (E1 - 1.0) : (type == 1 ? (1.0 - E1) : (c.template Et<ONSITE>(1, -s, pr) - E1));
      const double dE_own = sp == 0 ? dE0 : dE1;
      const double iem_slot = c.template iem1t<ONSITE>(sp, s, pr);
      iem_own = iem_slot;
      double* snn = snn2 + (i & 1);
      const bool hitR = spec_slot == slot && spec_r == r, hitA = specA_slot == slot && spec_r + 1 == r;
      const bool hit = spec_type == type && spec_jver == jver && (hitR || hitA);
      const int hbuf = (hitR ? 0 : specA_buf) * spec_stride;
      cp_async_wait_all();     // this thread's own copies of the previous proposal (long done; it reads only those)
      if (hit) {
        if (rl < r) {
          const int ja = Js[rl];
          const double raw = spec_own[hbuf + rl];
          if (role == 0) scol[rl] = x_from_raw(raw, ja == slot, slot < k0, iem_slot);      // X(ja, slot)
          else srow[rl] = x_from_raw(raw, ja == slot, ja < k0, jiem[rl]);                  // X(slot, ja)
        }
        if (tid == 0) {
          const double raw = spec_dg[hbuf];
          if (slot < k0 && type == 1) *snn = -raw * iem_slot;
          else *snn = 1.0 / dE_own + x_from_raw(raw, true, slot < k0, iem_slot);
        }
      } else {
        for (int a = rl; a < r; a += 256) {
          const int ja = Js[a];
          if (role == 0) scol[a] = X(ja, slot, iem_slot);
          else srow[a] = X(slot, ja, jiem[a]);
        }
        if (tid == 0) {
          if (slot < k0 && type == 1) *snn = -Ncur[(size_t)slot * ld + slot] * iem_slot;
          else *snn = 1.0 / dE_own + X(slot, slot, iem_slot);
        }
      }
      // copies of the next proposal, assuming this one is rejected, plus the entry for J[r] = this slot if it is accepted
      spec_slot = -1; specA_slot = -1; specA_buf = 0;
      if (i + 1 < win) {
        const NextSlots nx = next_slots(prop[i + 1], k0, kcur, live, type, slot, j);
        const int tn = nx.type, ns = nx.ns, nsA = nx.nsA;
        spec_type = tn; spec_r = r; spec_jver = jver;
        auto issue = [&](int nsl, int buf) {
          const double* coln = nsl < k0 ? Ncur + (size_t)nsl * ld : Gx + (size_t)(nsl - k0) * ld;
          if (rl <= r) {
            const int ja = rl < r ? Js[rl] : slot;
            const double* src = role == 0 ? coln + ja
                                          : (ja < k0 ? Ncur + (size_t)ja * ld + nsl : Gx + (size_t)(ja - k0) * ld + nsl);
            cp_async_8(spec_own + buf * spec_stride + rl, src);
          }
          if (tid == 0) cp_async_8(spec_dg + buf * spec_stride, coln + nsl);
        };
        if (ns >= 0) { spec_slot = ns; issue(ns, 0); }
        if (nsA >= 0) {
          specA_slot = nsA;
          if (nsA != ns) { specA_buf = 1; issue(nsA, 1); }
        }
      }
      __syncthreads();
      double part = 0.0, apart = 0.0;
      for (int a = row4; a < r; a += 64) {
        // lane q4 of a row takes the entries b = 16 i + 4 q4 + (0..3): with the odd leading dimension of S^-1 the 16 lanes
        // of a half-warp (4 rows x 4 lanes) then hit 16 different 8-byte banks for every one of the four loads (the
        // interleaved assignment b = 4 i + q4 put (row a, lane q) and (row a + 1, lane q - 1) on the same bank: the two
        // products were a third of the kernel's warp-state samples, MIO throttle and shared-memory scoreboard), and
        // the vector operand arrives as two 16-byte broadcast loads
        double s0 = 0.0, s1 = 0.0;
        if (!sinv_smem) {      // S^-1 in L2: the interleaved assignment keeps the four lanes of a row on one 32-byte sector
          int b = q4;
          if (role == 0) {
            const double* Sa = Sv + a;
            for (; b + 4 < r; b += 8) { s0 += Sa[(size_t)b * lds] * scol[b]; s1 += Sa[(size_t)(b + 4) * lds] * scol[b + 4]; }
            if (b < r) s0 += Sa[(size_t)b * lds] * scol[b];
          } else {
            const double* Sa = Sv + (size_t)a * lds;
            for (; b + 4 < r; b += 8) { s0 += srow[b] * Sa[b]; s1 += srow[b + 4] * Sa[b + 4]; }
            if (b < r) s0 += srow[b] * Sa[b];
          }
        } else if (role == 0) {
          const double* Sa = Sv + a;
          for (int b0 = 4 * q4; b0 < r; b0 += 16) {
            if (b0 + 3 < r) {
              const double2 v01 = *reinterpret_cast<const double2*>(scol + b0), v23 = *reinterpret_cast<const double2*>(scol + b0 + 2);
              s0 += Sa[(size_t)b0 * lds] * v01.x;       s1 += Sa[(size_t)(b0 + 1) * lds] * v01.y;
              s0 += Sa[(size_t)(b0 + 2) * lds] * v23.x; s1 += Sa[(size_t)(b0 + 3) * lds] * v23.y;
            } else {
              for (int b = b0; b < r; ++b) s0 += Sa[(size_t)b * lds] * scol[b];
            }
          }
        } else {
          const double* Sa = Sv + (size_t)a * lds;
          for (int b0 = 4 * q4; b0 < r; b0 += 16) {
            if (b0 + 3 < r) {
              const double2 v01 = *reinterpret_cast<const double2*>(srow + b0), v23 = *reinterpret_cast<const double2*>(srow + b0 + 2);
              s0 += v01.x * Sa[b0];     s1 += v01.y * Sa[b0 + 1];
              s0 += v23.x * Sa[b0 + 2]; s1 += v23.y * Sa[b0 + 3];
            } else {
              for (int b = b0; b < r; ++b) s0 += srow[b] * Sa[b];
            }
          }
        }
        double t = s0 + s1;
        t += __shfl_xor_sync(quad_mask, t, 1);
        t += __shfl_xor_sync(quad_mask, t, 2);
        if (q4 == 0) {
          if (role == 0) { tv[a] = t; part += srow[a] * t; apart += fabs(srow[a] * t); }
          else tpv[a] = t;
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        part += __shfl_xor_sync(0xffffffffu, part, o);
        apart += __shfl_xor_sync(0xffffffffu, apart, o);
      }
      if ((tid & 31) == 0) { red[tid >> 5] = part; red[16 + (tid >> 5)] = apart; }
      __syncthreads();
      double dot = 0.0, adot = 0.0;
#pragma unroll
      for (int q = 0; q < 8; ++q) { dot += red[q]; adot += red[16 + q]; }   // role-1 warps (8..15) hold zeros
      const double stil = *snn - dot;
      double o0[2], o1[2];
      exchange(stil, fabs(*snn) + adot, o0, o1);
      const double stil0 = o0[0], stil1 = o1[0];
      {
        // no division on the decision path: amp_s errlvl > guard  <=>  num_s errlvl > guard den_s
        const double den0 = fmax(fabs(stil0), 1e-300), den1 = fmax(fabs(stil1), 1e-300);
        if (r > 0 && (o0[1] * errlvl > c.guard_amp * den0 || o1[1] * errlvl > c.guard_amp * den1)) { guard_end = 1; break; }
        amp_n0 = o0[1]; amp_n1 = o1[1]; amp_d0 = den0; amp_d1 = den1;
      }
      stil_own = stil;
      R = pref * ((dE0 * stil0) * (dE1 * stil1));
      accept = pi.u < fabs(R);
    }
    if (tid == 0 && sp == 0 && log_count < (int64_t)c.log_capacity) {
      LogEntry e;
      e.p = p; e.type = type;
      e.arg = (type == 0) ? c.cfg_site[off_old + slot] : j;
      e.tau = (type == 0) ? c.cfg_tau[off_old + slot] : 0.0;
      e.spin = (type == 0) ? (int)spin_s[slot] : 0;
      e.accepted = accept ? 1 : 0;
      e.R = R; e.u = pi.u;
      c.log[(size_t)w * c.log_capacity + log_count] = e;
    }
    ++log_count;
    if (slot >= 0) {
      const double aR = fmax(fabs(R), 1e-300), du = fabs(pi.u - fabs(R));
      if (du * mm_aR < mm_du * aR) { mm_du = du; mm_aR = aR; }      // smallest du / aR, divided once at write-back
    }
    sum_k += (double)kcur;
    if (accept && type == 0 && kcur + 1 > c.max_k) { status = -2; break; }
    if (accept && down) {
      const double inv = 1.0 / stil_own;
      for (int a = tid; a < r; a += kClThreads) {
        tv[a] = Sv[a + (size_t)apos * lds];
        tpv[a] = Sv[apos + (size_t)a * lds];
      }
      __syncthreads();
      for (int a = tid & 63; a < r; a += 64) {
        const double ta = tv[a] * inv;
        double* Sa = Sv + a;
        for (int b = tid >> 6; b < r; b += 8) Sa[(size_t)b * lds] -= ta * tpv[b];
      }
      __syncthreads();
      const int last = r - 1;
      if (apos != last) {
        for (int b = tid; b < r; b += kClThreads) Sv[apos + (size_t)b * lds] = Sv[last + (size_t)b * lds];
        __syncthreads();
        for (int a = tid; a < last; a += kClThreads) Sv[a + (size_t)apos * lds] = Sv[a + (size_t)last * lds];
      }
      if (tid == 0 && apos != last) jiem[apos] = jiem[last];
      if (tid == 0) {
        jpos[slot - k0] = -1;
        if (apos != last) {
          const int moved = Js[last];
          Js[apos] = moved;
          if (moved >= k0) jpos[moved - k0] = apos;
        }
      }
      for (int idx = tid; idx < len - 1; idx += kClThreads) live_alt[idx] = live[idx + (idx >= j ? 1 : 0)];
      int* t = live; live = live_alt; live_alt = t;
      --len; --kcur; ++acc_rem;
      if (R < 0.0) sign = -sign;
      --r; ++jver;      // J was re-ordered: speculative loads of the next proposal are void
    } else if (accept) {
      const double inv = 1.0 / stil_own;
      for (int a = tid & 63; a < r; a += 64) {
        const double ta = tv[a] * inv;
        double* Sa = Sv + a;
        for (int b = tid >> 6; b < r; b += 8) Sa[(size_t)b * lds] += ta * tpv[b];
      }
      for (int a = tid; a < r; a += kClThreads) {
        Sv[a + (size_t)r * lds] = -tv[a] * inv;
        Sv[r + (size_t)a * lds] = -tpv[a] * inv;
      }
      if (tid == 0) { Sv[r + (size_t)r * lds] = inv; Js[r] = slot; jiem[r] = iem_own; }
      errlvl = fmax(errlvl, amp_n0 * amp_d1 > amp_n1 * amp_d0 ? amp_n0 / amp_d0 : amp_n1 / amp_d1);   // max of the two ratios, one division
      if (type == 0) {
        if (tid == 0) {
          live[len] = slot; jpos[slot - k0] = r;
          if (sp == 0) c.cfg_id[off_old + slot] = next_id;
        }
        ++len; ++kcur; ++next_id; ++acc_ins;
      } else if (type == 2) {
        if (tid == 0) flipped[slot] = 1;     // the vertex stays in the list; its spin changes at write-back
        ++acc_flip;
      } else {
        for (int idx = tid; idx < len - 1; idx += kClThreads) live_alt[idx] = live[idx + (idx >= j ? 1 : 0)];
        int* t = live; live = live_alt; live_alt = t;
        --len; --kcur; ++acc_rem;
      }
      if (R < 0.0) sign = -sign;
      ++r;
    }
    if (accept) __syncthreads();
    --props_left; ++p;
    if (props_left == 0) ++sweeps_done;
    if (r == c.delay) break;
  }
  __syncthreads();
  if (props_left == 0 && sweeps_left == 0) finished = true;

  // ---- write back.  Each CTA: its own S^-1.  Rank 0: list, maps, scalars.
  if (sinv_smem) {
    double* Sg = c.Sinv + ((size_t)w * 2 + sp) * (size_t)c.ldr * c.delay;
    for (int a = tid & 63; a < r; a += 64)
      for (int b = tid >> 6; b < r; b += 8) Sg[a + (size_t)b * c.ldr] = Sv[a + (size_t)b * lds];
  }
  cluster.sync();   // both CTAs are past every read of the walker state and of cfg_id before rank 0 rewrites them
  if (sp == 0) {
    int* rowmap = c.rowmap + (size_t)w * c.cap;
    for (int i = tid; i < kcur; i += kClThreads) {
      const int sl = live[i];
      rowmap[i] = sl;
      c.cfg_site[off_new + i] = c.cfg_site[off_old + sl];
      c.cfg_tau[off_new + i] = c.cfg_tau[off_old + sl];
      c.cfg_spin[off_new + i] = (sl < k0 && flipped[sl]) ? -c.cfg_spin[off_old + sl] : c.cfg_spin[off_old + sl];
      c.cfg_id[off_new + i] = c.cfg_id[off_old + sl];
    }
    for (int a = tid; a < r; a += kClThreads) c.J[(size_t)w * c.delay + a] = Js[a];
    if (tid == 0) {
      st.k_new = kcur;
      st.k = kcur;
      st.m = k0;
      st.cfg_cur = cfg_old ^ 1;
      st.r = r;
      st.n_src = n_cur0;
      st.n_cur = r > 0 ? (n_cur0 ^ 1) : n_cur0;
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
      atomicMax(c.n_active + 1, kcur);
      if (finished || status) {
        st.active = 0;
        atomicSub(c.n_active, 1);
      }
    }
  }
}

}  // namespace ctaux
