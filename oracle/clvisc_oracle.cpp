// CPU ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
// load this library.  It shares no code, header, table or helper with the CUDA path.
//
// Plain fp64 restatement of the CLVisc evolution step (arXiv:1802.04449), written from
// /root/reference/PAPER.md in the paper's order and notation, with the readings listed in
// DESIGN.md ("Readings", IDs A1..A25 from SURVEY.md section 8c):
//   * hydro equations in tilde variables      PAPER.md:123-183  (Eq.18-38)
//   * KT central scheme                       PAPER.md:193-213  (Eq.40-44)
//   * RK2 predictor/corrector with u* = 2u^n - u^{n-1}   PAPER.md:225-239 (Eq.49-54)
//   * root-find T_ideal = T - pi -> e, u      PAPER.md:229,235  (Eq.51,54)
// Pins (tests/test_oracle_*.py): ideal + Israel-Stewart Bjorken, Gubser (ideal closed form and
// IS ODE), exact conservation, brute-force per-cell evaluator on 4^3, root-find closed form,
// EoS closed form, mirror symmetry.  Unpinned conventions (shared rule, not shared code):
// A8 dynamic floor, A14 pi limiter, A23 bootstrap of u^{-1} -- "parity unpinned" for those.
//
// Notation: tilde/tetrad components, g~ = diag(1,-1,-1,-1); u~ = gamma(1,vx,vy,veta);
// frame tensor T_f^{mu nu} = (e+P)u~^mu u~^nu - P g~^{mu nu} + pi~^{mu nu};  paper's T~ = tau*T_f.
// Evolved: Q_T^mu = tau T_f^{tau mu}, Q_pi = u~^tau pi~^{mu nu}.
// pi component order: 0 tt, 1 tx, 2 ty, 3 tn, 4 xx, 5 xy, 6 xn, 7 yy, 8 yn, 9 nn.
// State per cell: e, u~^x, u~^y, u~^eta, pi~[10]; history u~^i at step n-1.
// No blocking, fusion or reordering beyond what the algorithm states; OpenMP only splits the
// flat cell loop.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>

namespace {

const double HBARC = 0.1973269804;  // GeV fm (A18)

// symmetric index map (mu,nu) -> 0..9
const int PIDX[4][4] = {{0, 1, 2, 3}, {1, 4, 5, 6}, {2, 5, 7, 8}, {3, 6, 8, 9}};
const double GMET[4] = {1.0, -1.0, -1.0, -1.0};  // g~ (Eq.23)

struct Eos {
  int kind = 0;  // 0 conformal, 1 table
  int n = 0;
  double e_min = 0, e_max = 0, c_sb = 0;
  std::vector<double> P, T;
  double node(int k) const { return e_min * std::pow(e_max / e_min, double(k) / double(n - 1)); }
};

// EoS: returns P, c_s^2, T at energy density e.  (A16, A17)
void eos_eval(const Eos& eos, double e, double* P, double* cs2, double* T) {
  if (eos.kind == 0) {  // EOSI
    *P = e / 3.0;
    *cs2 = 1.0 / 3.0;
    *T = HBARC * std::sqrt(std::sqrt(std::max(e, 0.0) / (eos.c_sb * HBARC)));
    return;
  }
  const int n = eos.n;
  if (e <= eos.e_min) {  // below the table: P linear through the origin, T ~ e^{1/4}
    *P = eos.P[0] * e / eos.e_min;
    *cs2 = eos.P[0] / eos.e_min;
    *T = eos.T[0] * std::sqrt(std::sqrt(std::max(e, 0.0) / eos.e_min));
    return;
  }
  if (e >= eos.e_max) {  // above: conformal continuation
    *P = eos.P[n - 1] + (e - eos.e_max) / 3.0;
    *cs2 = 1.0 / 3.0;
    *T = eos.T[n - 1] * std::sqrt(std::sqrt(e / eos.e_max));
    return;
  }
  double dln = std::log(eos.e_max / eos.e_min) / double(n - 1);
  int k = int(std::floor(std::log(e / eos.e_min) / dln));
  k = std::min(std::max(k, 0), n - 2);
  while (k > 0 && e < eos.node(k)) --k;
  while (k < n - 2 && e >= eos.node(k + 1)) ++k;
  double e0 = eos.node(k), e1 = eos.node(k + 1);
  double f = (e - e0) / (e1 - e0);
  *P = eos.P[k] + f * (eos.P[k + 1] - eos.P[k]);   // linear in e inside the bracket
  *cs2 = (eos.P[k + 1] - eos.P[k]) / (e1 - e0);    // slope of the segment
  *T = eos.T[k] + f * (eos.T[k + 1] - eos.T[k]);
}

double minmod3(double a, double b, double c) {
  if (a > 0 && b > 0 && c > 0) return std::min(a, std::min(b, c));
  if (a < 0 && b < 0 && c < 0) return std::max(a, std::max(b, c));
  return 0.0;
}

struct Oracle {
  int nx, ny, nz;
  double d[3];
  int bc[3];
  int geometry;  // 0 Milne, 1 Cartesian (all Christoffel terms 0)
  Eos eos;
  double dtau, tau0, eta_s;
  double theta = 1.1, e_floor = 1e-7, xi = 1.0, v_max = 1.0 - 1e-10;
  int strict_eq53 = 0;
  int step = 0;
  bool loaded = false;
  size_t N;
  // state n
  std::vector<double> e, u[3], pi[10], uprev[3];
  // counters
  long n_floor = 0, n_clamp = 0, n_limit = 0;
  double cfl[3] = {0, 0, 0}, e_max_seen = 0;

  size_t idx(int i, int j, int k) const { return (size_t(k) * ny + j) * nx + i; }
  // boundary rule a11: clamp (zero-gradient outflow) or wrap (periodic)
  int bmap(int a, int i) const {
    int n = (a == 0 ? nx : a == 1 ? ny : nz);
    if (bc[a] == 1) return ((i % n) + n) % n;
    return std::min(std::max(i, 0), n - 1);
  }
  size_t nb(int i, int j, int k, int a, int off) const {
    if (a == 0) return idx(bmap(0, i + off), j, k);
    if (a == 1) return idx(i, bmap(1, j + off), k);
    return idx(i, j, bmap(2, k + off));
  }
  bool viscous() const { return eta_s > 0.0; }
};

// A view of one state (e, u~^i, pi~) on the grid.
struct State {
  const double* e;
  const double* u[3];
  const double* pi[10];  // all null => ideal (pi == 0)
};

// Full frame tensor T_f^{mu nu} at one cell (Eq.1 :50 in tilde components, Eq.18-23).
void frame_tensor(const Oracle& o, const State& s, size_t c, bool use_pi, double P, double Tf[4][4],
                  double ut[4]) {
  double ux = s.u[0][c], uy = s.u[1][c], un = s.u[2][c];
  ut[0] = std::sqrt(1.0 + ux * ux + uy * uy + un * un);
  ut[1] = ux; ut[2] = uy; ut[3] = un;
  double e = s.e[c];
  for (int m = 0; m < 4; ++m)
    for (int n = 0; n < 4; ++n) {
      double t = (e + P) * ut[m] * ut[n];
      if (m == n) t -= P * GMET[m];
      if (use_pi) t += s.pi[PIDX[m][n]][c];
      Tf[m][n] = t;
    }
}

// Local maximum signal speed along axis a (A6; formula of Ref.[55]).
double signal_speed(double va, double v2, double cs2) {
  double cs = std::sqrt(cs2);
  double disc = (1.0 - v2) * (1.0 - v2 * cs2 - va * va * (1.0 - cs2));
  return (std::fabs(va) * (1.0 - cs2) + cs * std::sqrt(std::max(disc, 0.0))) / (1.0 - v2 * cs2);
}

// Workspace of per-point quantities for one RHS evaluation (steps 1-2 of SURVEY 8c).
struct PointTables {
  std::vector<double> P, cs2, T;
  std::vector<double> Q[14];
  std::vector<double> F[14];
  std::vector<double> c;
};

// KT numerical flux at the face between cells c1 and c2 for one field (Eq.41-44, A4, A5).
double kt_face(double theta, const std::vector<double>& Q, const std::vector<double>& F, double cface,
               size_t c0, size_t c1, size_t c2, size_t c3) {
  double mq1 = minmod3(theta * (Q[c1] - Q[c0]), 0.5 * (Q[c2] - Q[c0]), theta * (Q[c2] - Q[c1]));
  double mq2 = minmod3(theta * (Q[c2] - Q[c1]), 0.5 * (Q[c3] - Q[c1]), theta * (Q[c3] - Q[c2]));
  double mf1 = minmod3(theta * (F[c1] - F[c0]), 0.5 * (F[c2] - F[c0]), theta * (F[c2] - F[c1]));
  double mf2 = minmod3(theta * (F[c2] - F[c1]), 0.5 * (F[c3] - F[c1]), theta * (F[c3] - F[c2]));
  double Ql = Q[c1] + 0.5 * mq1, Qr = Q[c2] - 0.5 * mq2;   // Eq.44, Eq.43
  double Fl = F[c1] + 0.5 * mf1, Fr = F[c2] - 0.5 * mf2;   // A5
  return 0.5 * (Fr + Fl) - 0.5 * cface * (Qr - Ql);        // Eq.41-42
}

// RHS operator R(e, u~, d_tau u~, pi~; tau) -> S_T,tot[4], S_pi,tot[10]  (Eq.45-48).
// dtu[4]: arrays of d_tau u~^mu.  use_pi=false: ideal fluid (pi terms skipped, A15).
// cfl_out (optional, 3 values): max over cells of c_a*h/Delta_a.
void rhs(const Oracle& o, const State& s, bool use_pi, const std::vector<double>* dtu, double tau,
         std::vector<double>* ST, std::vector<double>* SP, double* cfl_out) {
  const size_t N = o.N;
  const int nf = use_pi ? 14 : 4;
  const bool milne = (o.geometry == 0);
  const double tf = milne ? tau : 1.0;  // Q_T = tau*T_f^{tau mu}; Cartesian: factor 1
  PointTables pt;
  pt.P.resize(N); pt.cs2.resize(N); pt.T.resize(N); pt.c.resize(N);
  for (int m = 0; m < nf; ++m) { pt.Q[m].resize(N); pt.F[m].resize(N); }
  for (int m = 0; m < 4; ++m) ST[m].assign(N, 0.0);
  if (use_pi) for (int m = 0; m < 10; ++m) SP[m].assign(N, 0.0);

  // step 1-2: EoS and conserved variables at every cell
#pragma omp parallel for
  for (size_t c = 0; c < N; ++c) {
    double Tf[4][4], ut[4];
    eos_eval(o.eos, s.e[c], &pt.P[c], &pt.cs2[c], &pt.T[c]);
    frame_tensor(o, s, c, use_pi, pt.P[c], Tf, ut);
    for (int m = 0; m < 4; ++m) pt.Q[m][c] = tf * Tf[0][m];
    if (use_pi) for (int m = 0; m < 10; ++m) pt.Q[4 + m][c] = ut[0] * s.pi[m][c];
  }

  // steps 2-5: per axis, fluxes F_a, signal speed c_a, KT divergence (Eq.40); order x, y, eta (A22)
  for (int a = 0; a < 3; ++a) {
    double cflmax = 0.0;
    const double scale = (a == 2 && milne) ? 1.0 / (tau * o.d[2]) : 1.0 / o.d[a];
#pragma omp parallel for reduction(max : cflmax)
    for (size_t c = 0; c < N; ++c) {
      double Tf[4][4], ut[4];
      frame_tensor(o, s, c, use_pi, pt.P[c], Tf, ut);
      for (int m = 0; m < 4; ++m) pt.F[m][c] = tf * Tf[a + 1][m];
      if (use_pi) for (int m = 0; m < 10; ++m) pt.F[4 + m][c] = ut[a + 1] * s.pi[m][c];
      double g = ut[0];
      double v2 = (ut[1] * ut[1] + ut[2] * ut[2] + ut[3] * ut[3]) / (g * g);
      pt.c[c] = signal_speed(ut[a + 1] / g, v2, pt.cs2[c]);
      cflmax = std::max(cflmax, pt.c[c] * o.dtau * scale);
    }
    if (cfl_out) cfl_out[a] = cflmax;
#pragma omp parallel for
    for (size_t c = 0; c < N; ++c) {
      int i = int(c % o.nx), j = int((c / o.nx) % o.ny), k = int(c / (size_t(o.nx) * o.ny));
      size_t m2 = o.nb(i, j, k, a, -2), m1 = o.nb(i, j, k, a, -1);
      size_t p1 = o.nb(i, j, k, a, +1), p2 = o.nb(i, j, k, a, +2);
      double cr = std::max(pt.c[c], pt.c[p1]);   // face i+1/2
      double cl = std::max(pt.c[m1], pt.c[c]);   // face i-1/2
      for (int m = 0; m < nf; ++m) {
        double Hr = kt_face(o.theta, pt.Q[m], pt.F[m], cr, m1, c, p1, p2);
        double Hl = kt_face(o.theta, pt.Q[m], pt.F[m], cl, m2, m1, c, p1);
        double div = -(Hr - Hl) * scale;
        if (m < 4) ST[m][c] += div; else SP[m - 4][c] += div;
      }
    }
  }

  // step 6-7: geometric source of T (Eq.31, sign A1), velocity gradients, IS source (Eq.33, A1, A2)
#pragma omp parallel for
  for (size_t c = 0; c < N; ++c) {
    int i = int(c % o.nx), j = int((c / o.nx) % o.ny), k = int(c / (size_t(o.nx) * o.ny));
    double Tf[4][4], ut[4];
    frame_tensor(o, s, c, use_pi, pt.P[c], Tf, ut);
    if (milne) {
      ST[0][c] += -Tf[3][3];   // S_T^tau  = -T_f^{eta eta}
      ST[3][c] += -Tf[0][3];   // S_T^eta  = -T_f^{tau eta}
    }
    if (!use_pi) continue;

    // grad[mu][nu] = nabla~_mu u~^nu  (Eq.22, Eq.24-26; A9 central differences, A10 time level)
    double grad[4][4];
    for (int n = 0; n < 4; ++n) grad[0][n] = dtu[n][c];
    for (int a = 0; a < 3; ++a) {
      size_t cm = o.nb(i, j, k, a, -1), cp = o.nb(i, j, k, a, +1);
      double inv = 1.0 / (2.0 * o.d[a]);
      if (a == 2 && milne) inv /= tau;
      double gp = std::sqrt(1.0 + s.u[0][cp] * s.u[0][cp] + s.u[1][cp] * s.u[1][cp] + s.u[2][cp] * s.u[2][cp]);
      double gm = std::sqrt(1.0 + s.u[0][cm] * s.u[0][cm] + s.u[1][cm] * s.u[1][cm] + s.u[2][cm] * s.u[2][cm]);
      grad[a + 1][0] = (gp - gm) * inv;
      for (int n = 0; n < 3; ++n) grad[a + 1][n + 1] = (s.u[n][cp] - s.u[n][cm]) * inv;
    }
    if (milne) {
      grad[3][0] += ut[3] / tau;   // Eq.25
      grad[3][3] += ut[0] / tau;   // Eq.26
    }
    double theta_exp = grad[0][0] + grad[1][1] + grad[2][2] + grad[3][3];
    double Du[4];
    for (int n = 0; n < 4; ++n) {
      Du[n] = 0.0;
      for (int m = 0; m < 4; ++m) Du[n] += ut[m] * grad[m][n];              // D~ = u~^lambda nabla~_lambda
    }
    double e = s.e[c], P = pt.P[c], T = pt.T[c];
    double inv_taupi = T / (5.0 * o.eta_s * HBARC);     // tau_pi = 5 eta_v/(T s)
    double etav_over_taupi = (e + P) / 5.0;             // eta_v/tau_pi = (e+P)/5
    auto pic = [&](int m, int n) { return s.pi[PIDX[m][n]][c]; };
    for (int m = 0; m < 4; ++m)
      for (int n = m; n < 4; ++n) {
        // sigma~^{mu nu}: expansion of Eq.5
        double sig = GMET[m] * grad[m][n] + GMET[n] * grad[n][m] - ut[m] * Du[n] - ut[n] * Du[m]
                     - (2.0 / 3.0) * ((m == n ? GMET[m] : 0.0) - ut[m] * ut[n]) * theta_exp;
        double p = pic(m, n);
        double src = -p * inv_taupi + etav_over_taupi * sig - p * theta_exp / 3.0;
        double contr = 0.0;
        for (int b = 0; b < 4; ++b) contr += (ut[m] * pic(n, b) + ut[n] * pic(m, b)) * GMET[b] * Du[b];
        src -= contr;
        if (milne) {
          src -= p * ut[0] / tau;
          double I = 0.0;   // Eq.35-38 in the general form (A2)
          if (m == 0) I += pic(3, n);
          if (m == 3) I += pic(0, n);
          if (n == 0) I += pic(m, 3);
          if (n == 3) I += pic(m, 0);
          src -= I * ut[3] / tau;
        }
        SP[PIDX[m][n]][c] += src;
      }
  }
}

// Root-find T_id^{tau mu} -> e, u~^i  (Eq.51/54; A7, A8).  M[4] = (M0, Mx, My, Meta).
void rootfind(Oracle& o, const double M[4], double* e_out, double u_out[3], long* nfloor, long* nclamp) {
  double M0 = M[0];
  if (!(M0 > o.e_floor)) {
    *e_out = o.e_floor; u_out[0] = u_out[1] = u_out[2] = 0.0; ++*nfloor;
    return;
  }
  double Mi[3] = {M[1], M[2], M[3]};
  double Mabs = std::sqrt(Mi[0] * Mi[0] + Mi[1] * Mi[1] + Mi[2] * Mi[2]);
  if (Mabs > o.v_max * M0) {
    double sc = o.v_max * M0 / Mabs;
    for (int a = 0; a < 3; ++a) Mi[a] *= sc;
    Mabs = o.v_max * M0; ++*nclamp;
  }
  // g(e) = M0 - M^2/(M0+P(e)) - e, strictly decreasing on [0, M0]; safeguarded Newton.
  double lo = 0.0, hi = M0, e = M0 - Mabs * Mabs / (M0 + M0 / 3.0);
  if (!(e >= lo && e <= hi)) e = 0.5 * (lo + hi);
  for (int it = 0; it < 200; ++it) {
    double P, cs2, T;
    eos_eval(o.eos, e, &P, &cs2, &T);
    double g = M0 - Mabs * Mabs / (M0 + P) - e;
    if (std::fabs(g) <= 1e-15 * M0) break;
    if (g > 0) lo = e; else hi = e;
    double dg = Mabs * Mabs * cs2 / ((M0 + P) * (M0 + P)) - 1.0;
    double en = e - g / dg;
    if (!(en > lo && en < hi)) en = 0.5 * (lo + hi);
    if (en == e) break;
    e = en;
  }
  if (e < o.e_floor) { e = o.e_floor; ++*nfloor; }
  double P, cs2, T;
  eos_eval(o.eos, e, &P, &cs2, &T);
  double v[3], v2 = 0;
  for (int a = 0; a < 3; ++a) { v[a] = Mi[a] / (M0 + P); v2 += v[a] * v[a]; }
  double gam = 1.0 / std::sqrt(1.0 - v2);
  for (int a = 0; a < 3; ++a) u_out[a] = gam * v[a];
  *e_out = e;
}

// pi limiter (A14; not in the paper, required by BASELINE.json configs[3]).
void limit_pi(const Oracle& o, double e, double pi[10], long* nlimit) {
  if (!(o.xi > 0)) return;
  double P, cs2, T;
  eos_eval(o.eos, e, &P, &cs2, &T);
  double pp = pi[0] * pi[0] - 2.0 * (pi[1] * pi[1] + pi[2] * pi[2] + pi[3] * pi[3]) + pi[4] * pi[4] +
              pi[7] * pi[7] + pi[9] * pi[9] + 2.0 * (pi[5] * pi[5] + pi[6] * pi[6] + pi[8] * pi[8]);
  double mag = std::sqrt(std::fabs(pp));
  double r = o.xi * std::sqrt(e * e + 3.0 * P * P) / std::max(mag, 1e-300);
  if (r < 1.0) { for (int m = 0; m < 10; ++m) pi[m] *= r; ++*nlimit; }
}
