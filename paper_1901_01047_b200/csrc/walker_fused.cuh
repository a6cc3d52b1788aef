// Fused small-k walker: S1 + S3 + S4 of whole sweeps in ONE kernel, one CTA per walker, both N_sigma
// resident in shared memory (configs 1-2: k ~ 10-80, where the seven-launch block step of the large
// configurations is pure launch latency; SURVEY.md section 8a "configs 1-3: many tiny problems").
//
// With N in shared memory the delayed block buys nothing, so every accepted move is applied at once
// (the delay is a performance knob only, Q19: the chain is identical):
//   insert v:  q_a = -g(a,v)(E_v - 1), p_b = -g(v,b)(E_b - 1), d = E_v - g00 (E_v - 1)
//              u = N q, w = p N, stilde = d - p.u  = det A'/det A            (rank-1 operation)
//              N' = [[N + u w^T / stilde, -u / stilde], [-w^T / stilde, 1 / stilde]]
//   remove j:  det A'/det A = N_jj;  N'_ab = N_ab - N_aj N_jb / N_jj, slot j dropped
// Vertices live in physical SLOTS (free slots are reused), `live[]` maps list position -> slot, so a
// removal moves no matrix data; the state is written back in list order when the kernel ends.
// The S5 rebuild stays on the batched LU kernels: the host ends the launch at the rebuild cadence.
// Shared memory holds `fcap` <= max_k slots; a walker whose order would exceed fcap (a rare upward
// fluctuation) SPILLS: it stops before that proposal, writes its state back with the sweeps / proposals
// it still owes, and the host finishes its sweeps on the delayed-block path (same chain).
#pragma once
#include "walker_state.cuh"

namespace ctaux {

constexpr int kFusedThreads = 256;
constexpr int kFusedGroup = 128;

struct FusedSmem {
  int N0, N1, q, p, u, w, colv, rowv, red, tau, site, spin, id, live, freel, total, lds;
};
__host__ __device__ inline FusedSmem fused_smem_layout(int cap) {
  FusedSmem L;
  L.lds = cap | 1;
  int o = 0;
  L.N0 = o; o += cap * L.lds * 8;
  L.N1 = o; o += cap * L.lds * 8;
  L.q = o; o += 2 * cap * 8;
  L.p = o; o += 2 * cap * 8;
  L.u = o; o += 2 * cap * 8;
  L.w = o; o += 2 * cap * 8;
  L.red = o; o += 2 * 4 * 8;
  L.tau = o; o += cap * 8;
  L.id = o; o += cap * 8;
  L.site = o; o += cap * 4;
  L.live = o; o += cap * 4;
  L.freel = o; o += cap * 4;
  L.spin = o; o += (cap + 15) / 16 * 16;
  L.colv = 0; L.rowv = 0;
  L.total = o;
  return L;
}

template <bool ONSITE>   // the on-site Hubbard model (one gamma, one site per vertex) or interacting pairs through the tables
__global__ void __launch_bounds__(kFusedThreads, 1) k_walk_fused(DevCtx c, int n_sweeps, int n_props, int fcap) {
  extern __shared__ __align__(16) unsigned char fsm[];
  const int wk = blockIdx.x, tid = threadIdx.x;
  WalkerState& st = c.ws[wk];
  if (st.status) return;
  const int cap = fcap;
  if (st.k > cap) {   // does not fit: the whole call goes to the delayed-block path
    if (tid == 0) { st.sweeps_left = n_sweeps; st.props_left = 0; st.active = 1; st.r = 0; atomicAdd(c.n_active, 1); }
    return;
  }
  const FusedSmem L = fused_smem_layout(cap);
  const int lds = L.lds;
  const int sp = tid / kFusedGroup, lt = tid % kFusedGroup;
  double* const Nup = reinterpret_cast<double*>(fsm + L.N0);
  double* const Ndn = reinterpret_cast<double*>(fsm + L.N1);
  double* const N = reinterpret_cast<double*>(fsm + L.N0) + (size_t)sp * cap * lds;   // N1 follows N0
  double* qv = reinterpret_cast<double*>(fsm + L.q) + sp * cap;
  double* pv = reinterpret_cast<double*>(fsm + L.p) + sp * cap;
  double* uv = reinterpret_cast<double*>(fsm + L.u) + sp * cap;
  double* wv = reinterpret_cast<double*>(fsm + L.w) + sp * cap;
  double* red = reinterpret_cast<double*>(fsm + L.red);  // [2 spins][4 warps]
  double* tau_s = reinterpret_cast<double*>(fsm + L.tau);
  uint64_t* id_s = reinterpret_cast<uint64_t*>(fsm + L.id);
  int* site_s = reinterpret_cast<int*>(fsm + L.site);
  int* live = reinterpret_cast<int*>(fsm + L.live);
  int* freel = reinterpret_cast<int*>(fsm + L.freel);
  signed char* spin_s = reinterpret_cast<signed char*>(fsm + L.spin);

  // ---- load: slot i = list position i
  int k = st.k;
  const size_t off = c.cfg_off(wk, st.cfg_cur);
  {
    const double* Ng = c.N(wk, sp, st.n_cur);
    for (int idx = lt; idx < cap * lds; idx += kFusedGroup) N[idx] = 0.0;
    __syncthreads();
    for (int idx = lt; idx < k * k; idx += kFusedGroup) {
      const int a = idx % k, b = idx / k;
      N[a + b * lds] = Ng[(size_t)b * c.ld + a];
    }
    for (int i = tid; i < k; i += kFusedThreads) {
      tau_s[i] = c.cfg_tau[off + i]; site_s[i] = c.cfg_site[off + i];
      spin_s[i] = (signed char)c.cfg_spin[off + i]; id_s[i] = c.cfg_id[off + i];
      live[i] = i;
    }
    for (int i = tid; i < cap - k; i += kFusedThreads) freel[i] = cap - 1 - i;  // stack: top = lowest free slot
  }
  int nfree = cap - k, hi = k;   // hi: slots in use are < hi
  uint64_t p = st.p, next_id = st.next_id;
  int sign = st.sign, status = 0, spill_sweeps = -1, spill_props = 0;
  int64_t acc_ins = 0, acc_rem = 0, acc_flip = 0, log_count = st.log_count;
  double mm_du = st.min_margin, mm_aR = 1.0, sum_k = 0.0;   // decision margin as a fraction (no division per proposal)
  int sweeps_done = 0;
  // site_s[] holds the PAIR index of every slot (= the site in the on-site model); E and the site a spin sector sees
  // come from the pair tables of DevCtx
  __syncthreads();

  if (n_props > 0) n_sweeps = 1;     // ctaux_propose: one partial sweep of exactly n_props proposals
  for (int sw = 0; sw < n_sweeps && !status; ++sw) {
    const int nprop = n_props > 0 ? n_props : (k > 16 ? k : 16);
    for (int ip = 0; ip < nprop; ++ip) {
      uint32_t wa[4], wb[4];
      philox4x32_10((uint32_t)(p & 0xffffffffu), (uint32_t)(p >> 32), 0u, 1u, st.key0, st.key1, wa);
      philox4x32_10((uint32_t)(p & 0xffffffffu), (uint32_t)(p >> 32), 1u, 1u, st.key0, st.key1, wb);
      const int type = c.flips ? (int)(((uint64_t)wb[2] * 3u) >> 32) : (int)(wa[0] & 1u);
      const double uu = unif53(wb[0], wb[1]);
      double R = 0.0;
      bool accept = false;
      int arg = -1, vs = 0, slot = -1, j = -1;
      double vtau = 0.0;
      double stil_own = 1.0;
      if (type == 0) {
        // ---------------------------------------------------------------- insertion
        vs = ((wa[0] >> 1) & 1u) ? -1 : +1;
        const int vsite = (int)(((uint64_t)wa[1] * (uint64_t)c.n_pairs) >> 32);   // pair index of the proposed vertex
        vtau = c.beta * unif53(wa[2], wa[3]);
        if (vtau >= c.beta) vtau = nextafter(c.beta, 0.0);
        arg = vsite;
        const double Ev1 = c.template Et<ONSITE>(sp, vs, vsite) - 1.0;          // E_v - 1
        const int vs_site = c.template sitet<ONSITE>(sp, vsite);                // the site this spin sector sees
        for (int a = lt; a < hi; a += kFusedGroup) {
          double qa = 0.0, pa = 0.0;
          const int sa = spin_s[a];
          if (sa != 0) {
            const double Ea1 = c.template Et<ONSITE>(sp, sa, site_s[a]) - 1.0;
            const int a_site = c.template sitet<ONSITE>(sp, site_s[a]);
            qa = -c.g(c.disp(a_site, vs_site), tau_s[a] - vtau) * Ev1;
            pa = -c.g(c.disp(vs_site, a_site), vtau - tau_s[a]) * Ea1;
          }
          qv[a] = qa; pv[a] = pa;
        }
        __syncthreads();
        // u = N q and w = p N: 64 rows x 2 roles when hi <= 64 (half 0 builds u, half 1 builds w), else one
        // thread per row builds both
        double part = 0.0;
        if (hi <= 64) {
          const int a = lt & 63, half = lt >> 6;
          if (a < hi) {
            double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
            int b = 0;
            if (half == 0) {
              const double* Na = N + a;
              for (; b + 3 < hi; b += 4) {
                s0 += Na[b * lds] * qv[b]; s1 += Na[(b + 1) * lds] * qv[b + 1];
                s2 += Na[(b + 2) * lds] * qv[b + 2]; s3 += Na[(b + 3) * lds] * qv[b + 3];
              }
              for (; b < hi; ++b) s0 += Na[b * lds] * qv[b];
              const double ua = (s0 + s1) + (s2 + s3);
              uv[a] = ua;
              part = pv[a] * ua;
            } else {
              const double* Na = N + a * lds;
              for (; b + 3 < hi; b += 4) {
                s0 += pv[b] * Na[b]; s1 += pv[b + 1] * Na[b + 1];
                s2 += pv[b + 2] * Na[b + 2]; s3 += pv[b + 3] * Na[b + 3];
              }
              for (; b < hi; ++b) s0 += pv[b] * Na[b];
              wv[a] = (s0 + s1) + (s2 + s3);
            }
          }
        } else {
          for (int a = lt; a < hi; a += kFusedGroup) {
            double s0 = 0.0, s1 = 0.0, t0 = 0.0, t1 = 0.0;
            int b = 0;
            for (; b + 1 < hi; b += 2) {
              s0 += N[a + b * lds] * qv[b];
              s1 += N[a + (b + 1) * lds] * qv[b + 1];
              t0 += pv[b] * N[b + a * lds];
              t1 += pv[b + 1] * N[b + 1 + a * lds];
            }
            if (b < hi) { s0 += N[a + b * lds] * qv[b]; t0 += pv[b] * N[b + a * lds]; }
            const double ua = s0 + s1;
            uv[a] = ua; wv[a] = t0 + t1;
            part += pv[a] * ua;
          }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        if ((tid & 31) == 0) red[sp * 4 + (lt >> 5)] = part;
        __syncthreads();
        const double e0 = c.template Et<ONSITE>(0, vs, vsite) - 1.0, e1 = c.template Et<ONSITE>(1, vs, vsite) - 1.0;   // E_v - 1 for spin up / down
        const double d0 = (e0 + 1.0) - c.g00 * e0;
        const double d1 = (e1 + 1.0) - c.g00 * e1;
        const double stil0 = d0 - ((red[0] + red[1]) + (red[2] + red[3]));
        const double stil1 = d1 - ((red[4] + red[5]) + (red[6] + red[7]));
        stil_own = sp == 0 ? stil0 : stil1;
        R = c.K / (double)(k + 1) * (stil0 * stil1);
        accept = uu < fabs(R);
        if (accept && k + 1 > c.max_k) { status = -2; accept = false; }
        if (accept && k + 1 > cap) {   // spill: this proposal is NOT consumed here
          spill_sweeps = n_sweeps - sw - 1; spill_props = nprop - ip;
          status = 1;
          __syncthreads();
          break;
        }
        if (accept) {
          slot = freel[nfree - 1];
          const double inv = 1.0 / stil_own;
          if (hi <= 64) {
            const int a = lt & 63;
            if (a < hi) {
              const double ua = uv[a] * inv;
              for (int b = lt >> 6; b < hi; b += 2) N[a + b * lds] += ua * wv[b];
            }
          } else {
            for (int a = lt; a < hi; a += kFusedGroup) {
              const double ua = uv[a] * inv;
              for (int b = 0; b < hi; ++b) N[a + b * lds] += ua * wv[b];
            }
          }
          __syncthreads();   // u, w fully consumed before the new row/column (slot may be < hi) is written
          for (int a = lt; a < hi; a += kFusedGroup) {
            N[a + slot * lds] = -uv[a] * inv;
            N[slot + a * lds] = -wv[a] * inv;
          }
          __syncthreads();
          if (lt == 0) N[slot + slot * lds] = inv;
          if (tid == 0) {
            tau_s[slot] = vtau; site_s[slot] = vsite; spin_s[slot] = (signed char)vs; id_s[slot] = next_id;
            live[k] = slot;
          }
          --nfree; ++k; ++next_id; ++acc_ins;
          if (slot >= hi) hi = slot + 1;
          if (R < 0.0) sign = -sign;
        }
      } else if (type == 2 && k > 0) {
        // ---------------------------------------------------------------- auxiliary-spin flip
        // column j of A changes by dE = E(-s) - E(s):  det A'/det A = 1 + dE (1 - N_jj)/(E - 1),
        // N' = N - (dE / ratio) x N_{j.},  x_a = (delta_aj - N_aj)/(E - 1)   (from N A = 1)
        j = (int)(((uint64_t)wa[1] * (uint64_t)k) >> 32);
        arg = j;
        slot = live[j];
        const int so = spin_s[slot];
        const int pr = site_s[slot];
        const double eo0 = c.template Et<ONSITE>(0, so, pr) - 1.0, en0 = c.template Et<ONSITE>(0, -so, pr) - 1.0;   // spin up: E(s) - 1, E(-s) - 1
        const double eo1 = c.template Et<ONSITE>(1, so, pr) - 1.0, en1 = c.template Et<ONSITE>(1, -so, pr) - 1.0;   // spin down
        const double n0 = Nup[slot + slot * lds], n1 = Ndn[slot + slot * lds];
        const double r0 = 1.0 + (en0 - eo0) * (1.0 - n0) / eo0;
        const double r1 = 1.0 + (en1 - eo1) * (1.0 - n1) / eo1;
        R = r0 * r1;
        accept = uu < fabs(R);
        if (accept) {
          const double f = sp == 0 ? (en0 - eo0) / (r0 * eo0) : (en1 - eo1) / (r1 * eo1);
          for (int a = lt; a < hi; a += kFusedGroup) {
            uv[a] = ((a == slot) ? 1.0 : 0.0) - N[a + slot * lds];
            wv[a] = N[slot + a * lds];
          }
          __syncthreads();
          if (hi <= 64) {
            const int a = lt & 63;
            if (a < hi) {
              const double ua = uv[a] * f;
              for (int b = lt >> 6; b < hi; b += 2) N[a + b * lds] -= ua * wv[b];
            }
          } else {
            for (int a = lt; a < hi; a += kFusedGroup) {
              const double ua = uv[a] * f;
              for (int b = 0; b < hi; ++b) N[a + b * lds] -= ua * wv[b];
            }
          }
          if (tid == 0) spin_s[slot] = (signed char)(-so);
          ++acc_flip;
          if (R < 0.0) sign = -sign;
        }
      } else if (type == 1 && k > 0) {
        // ---------------------------------------------------------------- removal
        j = (int)(((uint64_t)wa[1] * (uint64_t)k) >> 32);
        arg = j;
        slot = live[j];
        const double n0 = Nup[slot + slot * lds], n1 = Ndn[slot + slot * lds];
        R = (double)k / c.K * (n0 * n1);
        accept = uu < fabs(R);
        if (accept) {
          const double inv = 1.0 / (sp == 0 ? n0 : n1);
          for (int a = lt; a < hi; a += kFusedGroup) { uv[a] = N[a + slot * lds]; wv[a] = N[slot + a * lds]; }
          __syncthreads();
          if (hi <= 64) {
            const int a = lt & 63;
            if (a < hi) {
              const double ua = uv[a] * inv;
              for (int b = lt >> 6; b < hi; b += 2) N[a + b * lds] -= ua * wv[b];
            }
          } else {
            for (int a = lt; a < hi; a += kFusedGroup) {
              const double ua = uv[a] * inv;
              for (int b = 0; b < hi; ++b) N[a + b * lds] -= ua * wv[b];
            }
          }
          __syncthreads();
          for (int a = lt; a < hi; a += kFusedGroup) { N[a + slot * lds] = 0.0; N[slot + a * lds] = 0.0; }
          int lv = 0;
          if (tid > j && tid < k) lv = live[tid];                       // stable erase of list position j
          __syncthreads();
          if (tid > j && tid < k) live[tid - 1] = lv;
          if (tid == 0) { spin_s[slot] = 0; freel[nfree] = slot; }
          ++nfree; --k; ++acc_rem;
          if (R < 0.0) sign = -sign;
        }
      }
      if (tid == 0 && log_count < (int64_t)c.log_capacity) {
        LogEntry e;
        e.p = p; e.type = type; e.arg = arg;
        e.tau = type == 0 ? vtau : 0.0; e.spin = type == 0 ? vs : 0;
        e.accepted = accept ? 1 : 0; e.R = R; e.u = uu;
        c.log[(size_t)wk * c.log_capacity + log_count] = e;
      }
      ++log_count;
      if (type == 0 || arg >= 0) {
        const double aR = fmax(fabs(R), 1e-300), du = fabs(uu - fabs(R));
        if (du * mm_aR < mm_du * aR) { mm_du = du; mm_aR = aR; }      // smallest du / aR, divided once at write-back
      }
      sum_k += (double)(k - (accept ? (type == 0 ? 1 : (type == 1 ? -1 : 0)) : 0));   // k before the proposal
      ++p;
      __syncthreads();
      if (status) break;
    }
    if (!status) ++sweeps_done;
  }
  if (status == 1) status = 0;

  // ---- store: list order
  __syncthreads();
  {
    double* Ng = c.N(wk, sp, st.n_cur);
    for (int idx = lt; idx < k * k; idx += kFusedGroup) {
      const int a = idx % k, b = idx / k;
      Ng[(size_t)b * c.ld + a] = N[live[a] + live[b] * lds];
    }
    for (int i = tid; i < k; i += kFusedThreads) {
      const int sl = live[i];
      c.cfg_tau[off + i] = tau_s[sl]; c.cfg_site[off + i] = site_s[sl];
      c.cfg_spin[off + i] = (int)spin_s[sl]; c.cfg_id[off + i] = id_s[sl];
    }
  }
  if (tid == 0) {
    st.k = k; st.k_new = k; st.r = 0; st.m = 0; st.n_src = st.n_cur;
    st.next_id = next_id; st.p = p; st.sign = sign;
    st.acc_ins += acc_ins; st.acc_rem += acc_rem; st.acc_flip += acc_flip; st.sweeps += sweeps_done;
    st.blocks += sweeps_done; st.log_count = log_count;
    st.min_margin = mm_du / mm_aR; st.sum_k += sum_k;
    st.sweeps_left = 0; st.props_left = 0; st.active = 0;
    if (spill_sweeps >= 0) {
      st.sweeps_left = spill_sweeps; st.props_left = spill_props; st.active = 1;
      atomicAdd(c.n_active, 1);
    }
    if (status) st.status = status;
  }
}

}  // namespace ctaux
