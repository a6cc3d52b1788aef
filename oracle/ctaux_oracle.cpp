// ============================================================================
// CT-AUX walker ORACLE  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may build, link or call this file.  It shares no code, header, table or constant
// generator with paper_1901_01047_b200/csrc (the CUDA path).
//
// A plain, slow, single-threaded CPU implementation of the continuous-time
// auxiliary-field (CT-AUX) Monte-Carlo walker of arXiv:1901.01047 section 2.3
// (PAPER.md:166-228), written so that it can be checked against the paper by eye:
//
//   * Eq. (25) PAPER.md:194    cosh(gamma) = 1 + U beta Ncorr / (2K),  Ncorr = Nc
//   * Eq. (26)-(27) PAPER.md:198-201   weight of a configuration
//         (K / (2 beta Nc))^k  prod_sigma det A_sigma ,   A_sigma = N_sigma^{-1}
//   * PAPER.md:206             moves = vertex insertion / removal (rank-1 changes of N_sigma)
//   * BASELINE.json north_star N^{-1} = e^{-gamma sigma V} - G0 (e^{-gamma sigma V} - 1)
//
// Mode T0 (brute force, THE definition): every acceptance ratio is a quotient of
// determinants, each taken by LU with partial pivoting of the matrix built from scratch;
// N is the direct inverse of A built from the configuration.
// Mode T1 (textbook rank-1 / block-inverse updates, "rank-1 operations"):
// same chain, validated against T0 in tests, used where T0's O(k^3)-per-proposal cost is
// prohibitive.  N is re-inverted from scratch at the start of every sweep.
//
// Readings of points the paper leaves open are SURVEY.md section 8c Q1-Q31 / DESIGN.md:
//   Q1  table holds standard-sign G0 (<0 on (0,beta)); the matrix uses g = -G0
//   Q2  E(sigma, s) = exp(-gamma sigma s)
//   Q6  diagonal entry g(0, 0+)
//   Q7  equal times take the dtau >= 0 branch
//   Q8  M intervals, M+1 points, end points are the one-sided limits
//   Q11 1/2 insert, 1/2 remove      Q12 prefactors K/(k+1) and k/K
//   Q13 accept on |R|, carry sign   Q14 removal from empty: rejected, counter consumed
//   Q15 removal index = position in the ordered list; insert appends, erase is stable
//   Q16 sweep = max(16, k at sweep start) proposals       (convention: parity unpinned)
//   Q17 init_k Philox-drawn vertices accepted unconditionally (convention: parity unpinned)
//   Q29 uniform integers by multiply-shift (w * range) >> 32 (convention: parity unpinned)
//   NEXT-1 (off by default, orc_set_flips): auxiliary-spin flip as a third move, type = (w6*3)>>32, vertex at list
//       position (w1*k)>>32, R = prod_sigma det A'/det A.  Pinned by the Fock-space trace ratio, T1 == T0, and the
//       atomic-limit <k> with flips on; the word -> move mapping is a convention (parity unpinned).
//   NEXT-4 (off by default, orc_set_pairs): general density-density interaction between OPPOSITE spins, Eq. (19)-(21)
//       H_int = sum_p U_p [n_{a_p up} n_{b_p dn} - (n_{a_p up} + n_{b_p dn})/2] over N_corr pairs
//       p = (a_p, b_p, U_p) (on-site U: a = b; V between neighbours / layers / orbitals: a != b).  A
//       vertex is (p, tau, s); Eq. (24)-(25): cosh(gamma_p) = 1 + U_p beta N_corr / (2K); the up matrix sees site a_p,
//       the down matrix site b_p; both N_sigma stay k x k.  Vertex.site then holds the PAIR index.
//       Interactions between EQUAL spins (V', two rows of one N_sigma per vertex) are not covered.
// Pins (tests/test_oracle_*.py): closed-form table values, Fock-space trace = det A,
// one-vertex closed form, U->0 Poisson law, atomic-limit <k>, reversibility,
// permutation / spin symmetry, Philox against cuRAND's host generator, T1 == T0.
//
// Random numbers: Philox4x32-10 (Salmon et al., SC'11), re-stated here from the
// published algorithm; key = the walker's 64-bit seed, counter = (c0,c1,c2,c3).
// ============================================================================
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>

namespace {

// ---------------------------------------------------------------- Philox4x32-10
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   // multipliers
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   // Weyl key increments
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)M0 * c0;
    const uint64_t p1 = (uint64_t)M1 * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    const uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// 53-bit uniform in [0,1) from two words
double unif53(uint32_t a, uint32_t b) {
  const uint64_t u = ((uint64_t)a << 21) | (uint64_t)(b >> 11);
  return (double)u * (1.0 / 9007199254740992.0);  // 2^-53
}

// ---------------------------------------------------------------- dense helpers (row-major)
// LU with partial pivoting in place; returns sign of det, accumulates log|det|.
// A singular matrix returns sign 0.
int lu_inplace(std::vector<double>& a, int n, std::vector<int>& piv, double* logabs) {
  int sgn = 1;
  double la = 0.0;
  piv.resize(n);
  for (int c = 0; c < n; ++c) {
    int pr = c;
    double best = std::fabs(a[(size_t)c * n + c]);
    for (int r = c + 1; r < n; ++r) {
      const double v = std::fabs(a[(size_t)r * n + c]);
      if (v > best) { best = v; pr = r; }
    }
    piv[c] = pr;
    if (best == 0.0) { *logabs = -INFINITY; return 0; }
    if (pr != c) {
      for (int j = 0; j < n; ++j) std::swap(a[(size_t)c * n + j], a[(size_t)pr * n + j]);
      sgn = -sgn;
    }
    const double d = a[(size_t)c * n + c];
    if (d < 0) sgn = -sgn;
    la += std::log(std::fabs(d));
    for (int r = c + 1; r < n; ++r) {
      const double l = a[(size_t)r * n + c] / d;
      a[(size_t)r * n + c] = l;
      if (l != 0.0) {
        double* ar = &a[(size_t)r * n];
        const double* ac = &a[(size_t)c * n];
        for (int j = c + 1; j < n; ++j) ar[j] -= l * ac[j];
      }
    }
  }
  *logabs = la;
  return sgn;
}

// inverse via LU: solve A X = I column by column.  Returns false if singular.
bool invert(const std::vector<double>& A, int n, std::vector<double>& X) {
  std::vector<double> lu(A);
  std::vector<int> piv;
  double la;
  X.assign((size_t)n * n, 0.0);
  if (n == 0) return true;
  if (lu_inplace(lu, n, piv, &la) == 0) return false;
  // Work on B = P * I, row-major, all right-hand sides at once (rows of B are permuted unit rows).
  std::vector<double> B((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i) B[(size_t)i * n + i] = 1.0;
  for (int c = 0; c < n; ++c)
    if (piv[c] != c)
      for (int j = 0; j < n; ++j) std::swap(B[(size_t)c * n + j], B[(size_t)piv[c] * n + j]);
  // forward: L Y = B (unit lower)
  for (int i = 0; i < n; ++i) {
    double* bi = &B[(size_t)i * n];
    for (int l = 0; l < i; ++l) {
      const double f = lu[(size_t)i * n + l];
      if (f != 0.0) {
        const double* bl = &B[(size_t)l * n];
        for (int j = 0; j < n; ++j) bi[j] -= f * bl[j];
      }
    }
  }
  // backward: U X = Y
  for (int i = n - 1; i >= 0; --i) {
    double* bi = &B[(size_t)i * n];
    for (int l = i + 1; l < n; ++l) {
      const double f = lu[(size_t)i * n + l];
      if (f != 0.0) {
        const double* bl = &B[(size_t)l * n];
        for (int j = 0; j < n; ++j) bi[j] -= f * bl[j];
      }
    }
    const double d = lu[(size_t)i * n + i];
    for (int j = 0; j < n; ++j) bi[j] /= d;
  }
  X.swap(B);
  return true;
}

struct Vertex {
  uint64_t id;
  int32_t site;
  double tau;
  int32_t spin;  // auxiliary spin s = +1 / -1
};

struct LogEntry {   // 48 bytes, mirrored by numpy dtype in oracle/ctaux_oracle.py
  uint64_t p;       // proposal counter
  int32_t type;     // 0 insert, 1 remove
  int32_t arg;      // insert: site ; remove: list position j (-1 if k == 0)
  double tau;       // insert: proposed tau ; remove: 0
  int32_t spin;     // insert: proposed s ; remove: 0
  int32_t accepted;
  double R;         // signed acceptance ratio
  double u;         // uniform compared against |R|
};

struct Walker {
  // model
  int Lx, Ly, Nc, M;
  double beta, U, K;
  std::vector<double> table;  // [Nc][M+1], standard sign
  double egp, egm;            // e^{+gamma}, e^{-gamma}
  // NEXT-4: interacting pairs (empty = the on-site Hubbard model: pair p = site p, N_corr = Nc, one gamma)
  std::vector<int> pair_a, pair_b;
  std::vector<double> pair_egp;
  int n_corr() const { return pair_a.empty() ? Nc : (int)pair_a.size(); }
  int site_of(int sidx, int p) const { return pair_a.empty() ? p : (sidx == 0 ? pair_a[p] : pair_b[p]); }
  double tau_scale;           // M / beta
  // chain
  uint32_t key[2];
  std::vector<Vertex> L;
  uint64_t next_id = 0;
  uint64_t p = 0;
  int sign = 1;
  int mode = 0;  // 0 = T0, 1 = T1
  int flips = 0; // 1: auxiliary-spin FLIP as a third move (Fig. 5 (c)->(d)); SURVEY NEXT-1.
                 //    move type = (w6 * 3) >> 32: 0 insert, 1 remove, 2 flip, 1/3 each (w6 = reserved word wB[2]);
                 //    flip: vertex at list position (w1 * k) >> 32, s -> -s, R = prod_sigma det A'/det A
                 //    (symmetric proposal, no prefactor); k = 0: rejected.  0 (default): the two-move chain.
  int64_t acc_flip = 0;
  std::vector<LogEntry> log;
  int64_t acc_ins = 0, acc_rem = 0;
  double min_margin = INFINITY;
  // T0 cache: log|det A_sigma| and sign of the current configuration
  bool det_valid = false;
  double ld[2];
  int sd[2];
  // T1 state: N_sigma (k x k, row-major, stride k)
  std::vector<double> N[2];
  bool N_valid = false;

  // Eq. (25): cosh(gamma) = 1 + U beta Nc / (2K); e^{gamma} = c + sqrt(c^2 - 1)
  void set_gamma() {
    const double c = 1.0 + U * beta * (double)Nc / (2.0 * K);
    egp = c + std::sqrt(c * c - 1.0);
    egm = 1.0 / egp;
  }
  // E(sigma, s) = exp(-gamma sigma s): sigma = +1 (up, index 0) / -1 (down, index 1)
  double E(int sidx, int s, int p = 0) const {
    const int sigma = (sidx == 0) ? +1 : -1;
    const double eg = pair_a.empty() ? egp : pair_egp[p];
    return (sigma * s > 0) ? 1.0 / eg : eg;
  }
  // displacement index d(i,j) = ((xi-xj) mod Lx) + Lx ((yi-yj) mod Ly)
  int disp(int i, int j) const {
    const int xi = i % Lx, yi = i / Lx, xj = j % Lx, yj = j / Lx;
    const int dx = ((xi - xj) % Lx + Lx) % Lx;
    const int dy = ((yi - yj) % Ly + Ly) % Ly;
    return dx + Lx * dy;
  }
  // g(d, dtau) for dtau in (-beta, beta): positive-convention propagator by linear
  // interpolation in the table, antiperiodic in tau.
  double g(int d, double dtau) const {
    double sg = 1.0;
    if (dtau < 0.0) { sg = -1.0; dtau += beta; }
    const double x = dtau * tau_scale;
    int m = (int)std::floor(x);
    if (m > M - 1) m = M - 1;
    const double f = x - (double)m;
    const double* T = &table[(size_t)d * (M + 1)];
    return -sg * (T[m] + f * (T[m + 1] - T[m]));
  }
  double g_vv(int sidx, const Vertex& a, const Vertex& b, bool same) const {
    if (same) return -table[0];  // g(0, 0+)
    return g(disp(site_of(sidx, a.site), site_of(sidx, b.site)), a.tau - b.tau);
  }
  // A_sigma[i][j] = delta_ij E_j - g_ij (E_j - 1)
  void build_A(int sidx, const std::vector<Vertex>& V, std::vector<double>& A) const {
    const int n = (int)V.size();
    A.assign((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) {
        const double Ej = E(sidx, V[j].spin, V[j].site);
        const double gij = g_vv(sidx, V[i], V[j], i == j);
        A[(size_t)i * n + j] = (i == j ? Ej : 0.0) - gij * (Ej - 1.0);
      }
  }
  int logdet(int sidx, const std::vector<Vertex>& V, double* la) const {
    std::vector<double> A;
    std::vector<int> piv;
    build_A(sidx, V, A);
    if (V.empty()) { *la = 0.0; return 1; }
    return lu_inplace(A, (int)V.size(), piv, la);
  }
  void refresh_det() {
    if (det_valid) return;
    for (int s = 0; s < 2; ++s) sd[s] = logdet(s, L, &ld[s]);
    det_valid = true;
  }
  bool refresh_N() {
    bool ok = true;
    for (int s = 0; s < 2; ++s) {
      std::vector<double> A;
      build_A(s, L, A);
      ok = invert(A, (int)L.size(), N[s]) && ok;
    }
    N_valid = true;
    return ok;
  }

  Vertex draw_vertex(const uint32_t w[4]) const {
    Vertex v;
    v.id = 0;
    v.spin = ((w[0] >> 1) & 1u) ? -1 : +1;
    v.site = (int32_t)(((uint64_t)w[1] * (uint64_t)n_corr()) >> 32);   // site of the on-site model, pair index in general
    v.tau = beta * unif53(w[2], w[3]);
    if (v.tau >= beta) v.tau = std::nextafter(beta, 0.0);
    return v;
  }

  void reset(int init_k) {
    L.clear();
    for (int i = 0; i < init_k; ++i) {
      const uint32_t ctr[4] = {(uint32_t)i, 0u, 0u, 0u};
      uint32_t w[4];
      philox4x32_10(ctr, key, w);
      Vertex v = draw_vertex(w);
      v.id = (uint64_t)i;
      L.push_back(v);
    }
    next_id = (uint64_t)init_k;
    p = 0;
    det_valid = false;
    N_valid = false;
    refresh_det();
    sign = sd[0] * sd[1];
    log.clear();
    acc_ins = acc_rem = 0; acc_flip = 0;
    min_margin = INFINITY;
  }

  // product over sigma of det A'_sigma / det A_sigma, brute force (T0)
  double ratio_T0(const std::vector<Vertex>& Lnew) {
    refresh_det();
    double r = 1.0;
    for (int s = 0; s < 2; ++s) {
      double la;
      const int sg = logdet(s, Lnew, &la);
      if (sg == 0 || sd[s] == 0) return 0.0;
      r *= (double)(sg * sd[s]) * std::exp(la - ld[s]);
    }
    return r;
  }

  // ---- T1: insertion of v as last row/column.  A' = [[A, q], [p^T, d]]
  //   q_i = -g(i,v) (E_v - 1),  p_j = -g(v,j) (E_j - 1),  d = E_v - g(0,0+) (E_v - 1)
  //   det A'/det A = d - p^T N q
  struct InsWork { std::vector<double> Nq[2], pN[2]; double stilde[2]; };
  double ratio_ins_T1(const Vertex& v, InsWork& W) {
    const int k = (int)L.size();
    double r = 1.0;
    for (int s = 0; s < 2; ++s) {
      const double Ev = E(s, v.spin, v.site);
      std::vector<double> q(k), pr(k);
      for (int i = 0; i < k; ++i) {
        q[i] = -g_vv(s, L[i], v, false) * (Ev - 1.0);
        pr[i] = -g_vv(s, v, L[i], false) * (E(s, L[i].spin, L[i].site) - 1.0);
      }
      const double d = Ev - (-table[0]) * (Ev - 1.0);
      W.Nq[s].assign(k, 0.0);
      W.pN[s].assign(k, 0.0);
      const std::vector<double>& Ns = N[s];
      for (int i = 0; i < k; ++i) {
        const double* row = &Ns[(size_t)i * k];
        double acc = 0.0;
        for (int j = 0; j < k; ++j) acc += row[j] * q[j];
        W.Nq[s][i] = acc;
      }
      for (int i = 0; i < k; ++i) {
        const double* row = &Ns[(size_t)i * k];
        const double pi = pr[i];
        double* out = W.pN[s].data();
        for (int j = 0; j < k; ++j) out[j] += pi * row[j];
      }
      double dot = 0.0;
      for (int i = 0; i < k; ++i) dot += pr[i] * W.Nq[s][i];
      W.stilde[s] = d - dot;
      r *= W.stilde[s];
    }
    return r;
  }
  void apply_ins_T1(const InsWork& W) {
    const int k = (int)L.size();  // size BEFORE the insertion
    for (int s = 0; s < 2; ++s) {
      const double st = W.stilde[s];
      std::vector<double> Nn((size_t)(k + 1) * (k + 1));
      for (int i = 0; i < k; ++i) {
        const double f = W.Nq[s][i] / st;
        const double* row = &N[s][(size_t)i * k];
        double* out = &Nn[(size_t)i * (k + 1)];
        for (int j = 0; j < k; ++j) out[j] = row[j] + f * W.pN[s][j];
        out[k] = -f;
      }
      double* last = &Nn[(size_t)k * (k + 1)];
      for (int j = 0; j < k; ++j) last[j] = -W.pN[s][j] / st;
      last[k] = 1.0 / st;
      N[s].swap(Nn);
    }
  }
  // ---- T1: removal of list position j: det A'/det A = N_jj ; N'_ab = N_ab - N_aj N_jb / N_jj
  double ratio_rem_T1(int j) const {
    const int k = (int)L.size();
    return N[0][(size_t)j * k + j] * N[1][(size_t)j * k + j];
  }
  // flip of vertex j changes column j of A only: A' = A + dE (e_j - g_{.j}) e_j^T, dE = E'_j - E_j, and
  // N (e_j - g_{.j}) = (e_j - N_{.j}) / (E_j - 1)  (from N A = 1), so per spin
  //   det A'/det A = 1 + dE (1 - N_jj)/(E_j - 1),   N' = N - (dE / ratio) x_j N_{j.},  x_j[i] = (delta_ij - N_ij)/(E_j - 1)
  double ratio_flip_T1(int j, double r[2]) const {
    const int k = (int)L.size();
    for (int s = 0; s < 2; ++s) {
      const double Eo = E(s, L[j].spin, L[j].site), En = E(s, -L[j].spin, L[j].site);
      r[s] = 1.0 + (En - Eo) * (1.0 - N[s][(size_t)j * k + j]) / (Eo - 1.0);
    }
    return r[0] * r[1];
  }
  void apply_flip_T1(int j, const double r[2]) {
    const int k = (int)L.size();
    for (int s = 0; s < 2; ++s) {
      const double Eo = E(s, L[j].spin, L[j].site), En = E(s, -L[j].spin, L[j].site);
      const double f = (En - Eo) / r[s] / (Eo - 1.0);
      std::vector<double>& Nm = N[s];
      std::vector<double> x(k), row(k);
      for (int i = 0; i < k; ++i) { x[i] = ((i == j) ? 1.0 : 0.0) - Nm[(size_t)i * k + j]; row[i] = Nm[(size_t)j * k + i]; }
      for (int a = 0; a < k; ++a)
        for (int b = 0; b < k; ++b) Nm[(size_t)a * k + b] -= f * x[a] * row[b];
    }
  }
  void apply_rem_T1(int j) {
    const int k = (int)L.size();  // size BEFORE the removal
    for (int s = 0; s < 2; ++s) {
      const std::vector<double>& No = N[s];
      const double njj = No[(size_t)j * k + j];
      std::vector<double> Nn((size_t)(k - 1) * (k - 1));
      for (int a = 0, an = 0; a < k; ++a) {
        if (a == j) continue;
        const double f = No[(size_t)a * k + j] / njj;
        const double* row = &No[(size_t)a * k];
        const double* rj = &No[(size_t)j * k];
        double* out = &Nn[(size_t)an * (k - 1)];
        for (int b = 0, bn = 0; b < k; ++b) {
          if (b == j) continue;
          out[bn++] = row[b] - f * rj[b];
        }
        ++an;
      }
      N[s].swap(Nn);
    }
  }

  void propose_once() {
    const uint32_t plo = (uint32_t)(p & 0xffffffffu), phi = (uint32_t)(p >> 32);
    const uint32_t cA[4] = {plo, phi, 0u, 1u}, cB[4] = {plo, phi, 1u, 1u};
    uint32_t wA[4], wB[4];
    philox4x32_10(cA, key, wA);
    philox4x32_10(cB, key, wB);
    const int k = (int)L.size();
    LogEntry e;
    std::memset(&e, 0, sizeof(e));
    e.p = p;
    e.type = flips ? (int32_t)(((uint64_t)wB[2] * 3u) >> 32) : (int32_t)(wA[0] & 1u);
    e.u = unif53(wB[0], wB[1]);
    double R = 0.0;
    if (mode == 1 && !N_valid) refresh_N();
    if (e.type == 0) {
      Vertex v = draw_vertex(wA);
      e.arg = v.site; e.tau = v.tau; e.spin = v.spin;
      InsWork W;
      double prod;
      if (mode == 0) {
        std::vector<Vertex> Ln(L);
        Ln.push_back(v);
        prod = ratio_T0(Ln);
      } else {
        prod = ratio_ins_T1(v, W);
      }
      R = K / (double)(k + 1) * prod;
      e.accepted = (e.u < std::fabs(R)) ? 1 : 0;
      if (e.accepted) {
        if (mode == 1) apply_ins_T1(W);
        v.id = next_id++;
        L.push_back(v);
        det_valid = false;
        ++acc_ins;
      }
    } else if (e.type == 2) {
      if (k == 0) {
        e.arg = -1;
        R = 0.0;
        e.accepted = 0;
      } else {
        const int j = (int)(((uint64_t)wA[1] * (uint64_t)k) >> 32);
        e.arg = j;
        double r[2] = {1.0, 1.0};
        if (mode == 0) {
          std::vector<Vertex> Ln(L);
          Ln[j].spin = -Ln[j].spin;
          R = ratio_T0(Ln);
        } else {
          R = ratio_flip_T1(j, r);
        }
        e.accepted = (e.u < std::fabs(R)) ? 1 : 0;
        if (e.accepted) {
          if (mode == 1) apply_flip_T1(j, r);
          L[j].spin = -L[j].spin;
          det_valid = false;
          ++acc_flip;
        }
      }
    } else {
      if (k == 0) {
        e.arg = -1;
        R = 0.0;
        e.accepted = 0;
      } else {
        const int j = (int)(((uint64_t)wA[1] * (uint64_t)k) >> 32);
        e.arg = j;
        double prod;
        if (mode == 0) {
          std::vector<Vertex> Ln(L);
          Ln.erase(Ln.begin() + j);
          prod = ratio_T0(Ln);
        } else {
          prod = ratio_rem_T1(j);
        }
        R = (double)k / K * prod;
        e.accepted = (e.u < std::fabs(R)) ? 1 : 0;
        if (e.accepted) {
          if (mode == 1) apply_rem_T1(j);
          L.erase(L.begin() + j);
          det_valid = false;
          ++acc_rem;
        }
      }
    }
    if (e.accepted && R < 0.0) sign = -sign;
    e.R = R;
    const double aR = std::fabs(R);
    const double margin = std::fabs(e.u - aR) / std::max(aR, 1e-300);
    if (!(e.type != 0 && k == 0) && margin < min_margin) min_margin = margin;
    log.push_back(e);
    ++p;
  }

  void sweep(int n_sweeps) {
    for (int s = 0; s < n_sweeps; ++s) {
      if (mode == 1) refresh_N();  // T1: from-scratch inverse every sweep
      const int64_t n_prop = std::max<int64_t>(16, (int64_t)L.size());
      for (int64_t i = 0; i < n_prop; ++i) propose_once();
    }
  }
};

}  // namespace

// ============================================================================ C interface (ctypes)
extern "C" {

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  philox4x32_10(ctr, key, out);
}
double orc_unif53(uint32_t a, uint32_t b) { return unif53(a, b); }

void* orc_create(int Lx, int Ly, double beta, double U, double K, int M, const double* table,
                 uint64_t seed, int mode) {
  Walker* w = new Walker();
  w->Lx = Lx; w->Ly = Ly; w->Nc = Lx * Ly; w->M = M;
  w->beta = beta; w->U = U; w->K = K;
  w->table.assign(table, table + (size_t)w->Nc * (M + 1));
  w->tau_scale = (double)M / beta;
  w->set_gamma();
  w->key[0] = (uint32_t)(seed & 0xffffffffu);
  w->key[1] = (uint32_t)(seed >> 32);
  w->mode = mode;
  return w;
}
void orc_destroy(void* h) { delete (Walker*)h; }
void orc_reset(void* h, int init_k) { ((Walker*)h)->reset(init_k); }
// NEXT-4: interacting pairs (a_p up, b_p down, U_p).  gamma_p from Eq. (25) with N_corr = n_pairs.  n_pairs = 0 restores
// the on-site model.  Call before reset / set_state.
void orc_set_pairs(void* h, int n_pairs, const int32_t* a, const int32_t* b, const double* U) {
  Walker* w = (Walker*)h;
  w->pair_a.assign(a, a + n_pairs);
  w->pair_b.assign(b, b + n_pairs);
  w->pair_egp.resize(n_pairs);
  for (int p = 0; p < n_pairs; ++p) {
    const double c = 1.0 + U[p] * w->beta * (double)n_pairs / (2.0 * w->K);
    w->pair_egp[p] = c + std::sqrt(c * c - 1.0);
  }
  w->det_valid = false; w->N_valid = false;
}
double orc_pair_exp_gamma(void* h, int p) { return ((Walker*)h)->pair_egp[p]; }
void orc_set_flips(void* h, int on) { ((Walker*)h)->flips = on ? 1 : 0; }
int64_t orc_acc_flip(void* h) { return ((Walker*)h)->acc_flip; }
void orc_set_mode(void* h, int mode) { Walker* w = (Walker*)h; w->mode = mode; w->N_valid = false; w->det_valid = false; }

// Start from a given configuration (list order), proposal counter and next id.
void orc_set_state(void* h, int k, const uint64_t* id, const int32_t* site, const double* tau,
                   const int8_t* spin, uint64_t next_id, uint64_t p) {
  Walker* w = (Walker*)h;
  w->L.clear();
  for (int i = 0; i < k; ++i) {
    Vertex v; v.id = id ? id[i] : (uint64_t)i; v.site = site[i]; v.tau = tau[i]; v.spin = spin[i];
    w->L.push_back(v);
  }
  w->next_id = next_id; w->p = p;
  w->det_valid = false; w->N_valid = false;
  w->refresh_det();
  w->sign = w->sd[0] * w->sd[1];
  w->log.clear();
  w->acc_ins = w->acc_rem = 0;
  w->acc_flip = 0;
  w->min_margin = INFINITY;
}
void orc_sweep(void* h, int n_sweeps) { ((Walker*)h)->sweep(n_sweeps); }
void orc_propose(void* h, int64_t n) { Walker* w = (Walker*)h; for (int64_t i = 0; i < n; ++i) w->propose_once(); }

int orc_k(void* h) { return (int)((Walker*)h)->L.size(); }
int orc_sign(void* h) { return ((Walker*)h)->sign; }
uint64_t orc_p(void* h) { return ((Walker*)h)->p; }
uint64_t orc_next_id(void* h) { return ((Walker*)h)->next_id; }
int64_t orc_acc_ins(void* h) { return ((Walker*)h)->acc_ins; }
int64_t orc_acc_rem(void* h) { return ((Walker*)h)->acc_rem; }
double orc_min_margin(void* h) { return ((Walker*)h)->min_margin; }
double orc_exp_gamma(void* h) { return ((Walker*)h)->egp; }

void orc_get_config(void* h, uint64_t* id, int32_t* site, double* tau, int8_t* spin) {
  Walker* w = (Walker*)h;
  for (size_t i = 0; i < w->L.size(); ++i) {
    id[i] = w->L[i].id; site[i] = w->L[i].site; tau[i] = w->L[i].tau; spin[i] = (int8_t)w->L[i].spin;
  }
}
// A_sigma of the current configuration, row-major k x k.
void orc_get_A(void* h, int sidx, double* out) {
  Walker* w = (Walker*)h;
  std::vector<double> A;
  w->build_A(sidx, w->L, A);
  std::copy(A.begin(), A.end(), out);
}
// A_sigma of a GIVEN vertex list (row-major k x k); the walker's own state is not touched.  Accessor for the
// log-replay checks of the tests (determinants then taken by LAPACK): same build_A as everywhere else.
void orc_build_A(void* h, int sidx, int k, const int32_t* site, const double* tau, const int8_t* spin, double* out) {
  const Walker* w = (const Walker*)h;
  std::vector<Vertex> V((size_t)k);
  for (int i = 0; i < k; ++i) { V[i].id = (uint64_t)i; V[i].site = site[i]; V[i].tau = tau[i]; V[i].spin = spin[i]; }
  std::vector<double> A;
  w->build_A(sidx, V, A);
  std::copy(A.begin(), A.end(), out);
}
// N_sigma = A_sigma^{-1} by DIRECT inversion (the definition), row-major. Returns 0 ok, -1 singular.
int orc_get_N(void* h, int sidx, double* out) {
  Walker* w = (Walker*)h;
  std::vector<double> A, X;
  w->build_A(sidx, w->L, A);
  if (!invert(A, (int)w->L.size(), X)) return -1;
  std::copy(X.begin(), X.end(), out);
  return 0;
}
// T1's incrementally updated N (row-major); only meaningful in mode 1 after at least one proposal.
int orc_get_N_incremental(void* h, int sidx, double* out) {
  Walker* w = (Walker*)h;
  if (w->mode != 1 || !w->N_valid) return -1;
  std::copy(w->N[sidx].begin(), w->N[sidx].end(), out);
  return 0;
}
// log|det A_sigma| and its sign for the current configuration (brute force).
double orc_logdet(void* h, int sidx, int* sgn) {
  Walker* w = (Walker*)h;
  double la;
  *sgn = w->logdet(sidx, w->L, &la);
  return la;
}
// interpolated propagator g(d, dtau)
double orc_g(void* h, int d, double dtau) { return ((Walker*)h)->g(d, dtau); }

int64_t orc_log_size(void* h) { return (int64_t)((Walker*)h)->log.size(); }
void orc_get_log(void* h, void* out, int64_t first, int64_t count) {
  Walker* w = (Walker*)h;
  std::memcpy(out, w->log.data() + first, (size_t)count * sizeof(LogEntry));
}
void orc_clear_log(void* h) { ((Walker*)h)->log.clear(); }
int orc_log_entry_bytes() { return (int)sizeof(LogEntry); }

}  // extern "C"
