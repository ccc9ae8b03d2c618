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
// Pins (tests/test_oracle_*.py): ideal + Israel-Stewart Bjorken, Gubser (ideal closed form and IS ODE, to tau = 4
// against the survey's independent probe numbers), exact conservation, brute-force per-cell evaluator on 4^3,
// root-find closed form, EoS closed form, mirror symmetry, Riemann fan; the Milne terms that need u~^eta != 0
// (Eq.24-26, 31, 35-38) by a Minkowski-static fluid, a slice-uniform shear tensor and the Poincare-shifted Gubser
// PDE residual (test_oracle_milne_pins.py); the pi limiter (A14) by its invariant, the bootstrap of u^{-1} (A23)
// against ideal Gubser at O(h^2), strict Eq.53 (A12) and the printed Heun form (A26) by convergence / difference
// (test_oracle_limiter_bootstrap.py).  Still a shared convention without an external pin: the value of the
// dynamic floor (A8) -- "parity unpinned" for that one rule.
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
  int heun_printed = 0;   // A26: 0 = Shu-Osher bookkeeping (default), 1 = Eq.52-53 exactly as printed
  // the lambda_1 term of Eq.4 / Eq.33 and a free relaxation-time coefficient,
  //   tau_pi = c_tau eta_v/(T s)   (paper: c_tau = 5),   lambda_1 = lambda1_hat / e
  // needed by the paper's closed-form Gubser test (L = 2, eta_v/s = 0.2, lambda1_hat = -10 and
  // tau_pi from eta_hat lambda1_hat^2 = 3 tau_pi_hat, i.e. c_tau = 4 lambda1_hat^2 / 9).
  double lambda1_hat = 0.0, c_tau = 5.0;
  // SURVEY 8(f)-3 (PAPER.md:46-56 Eq.1-3; :153-171 Eq.28, 30, 32, 34; :614 "2 components in N and Pi": the 16-word cell):
  // bulk pressure Pi and net-baryon density n (local rest frame), evolved when ext = 1 (viscous runs only).
  //   A28  T_f^{mu nu} = (e + P + Pi) u~^mu u~^nu - (P + Pi) g~^{mu nu} + pi~^{mu nu}                    (Eq.1, :50)
  //   A29  S_Pi,tot = S_KT - (Pi + zeta theta~)/tau_Pi - Pi theta~/3 - u~^tau Pi / tau: Eq.3 (:56), the defining equation,
  //        written as a balance law, d_mu(u^mu Pi) = D Pi + Pi theta with D Pi = -(Pi + zeta theta)/tau_Pi - 4/3 Pi theta;
  //        the printed Eq.34 has +zeta theta~ (against Eq.3 and against the Navier-Stokes limit Pi = -zeta theta) and lacks
  //        the Milne term u~^tau Pi / tau that its shear twin Eq.33 carries (sign as A1)
  //   A30  zeta = (zeta/s) s with s = (e+P)/T and a constant zeta/s; tau_Pi = tau_pi (the paper leaves both open, :72)
  //   A31  N~^mu = tau n u~^mu (Eq.21, :128), S_N = 0 (Eq.32): Q_N = tau n u~^tau, F_a = tau n u~^a; n = Q_N/(tau u~^tau)
  //        after the root-find; the EoS does not depend on n (P(e) tables, :253-259)
  //   A32  the root-find carries Pi through the total pressure P_tot(e) = max(P(e) + Pi, 0) (continuous, non-decreasing:
  //        the root stays unique and |v| <= v_max): e = M0 - M^2/(M0 + P_tot), v = M/(M0 + P_tot); afterwards |Pi| <= xi P(e)
  //        (same xi as the pi limiter) -- a convention in the spirit of A14, "parity unpinned" beyond its invariant
  int ext = 0;
  double zeta_s = 0.0;
  std::vector<double> Pi, nB;
  long n_bulk_limit = 0;
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
  const double* Pi = nullptr;   // 8(f)-3: bulk pressure (null => 0) and net-baryon density (null => not evolved)
  const double* nB = nullptr;
};

// Full frame tensor T_f^{mu nu} at one cell (Eq.1 :50 in tilde components, Eq.18-23).
void frame_tensor(const Oracle& o, const State& s, size_t c, bool use_pi, double P, double Tf[4][4],
                  double ut[4]) {
  double ux = s.u[0][c], uy = s.u[1][c], un = s.u[2][c];
  ut[0] = std::sqrt(1.0 + ux * ux + uy * uy + un * un);
  ut[1] = ux; ut[2] = uy; ut[3] = un;
  double e = s.e[c];
  if (s.Pi) P += s.Pi[c];       // A28: the bulk pressure adds to the equilibrium pressure in T_f
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
  std::vector<double> Q[16];
  std::vector<double> F[16];
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
// SX (optional, with s.Pi / s.nB set): S_Pi,tot and S_N,tot (8(f)-3).
void rhs(const Oracle& o, const State& s, bool use_pi, const std::vector<double>* dtu, double tau,
         std::vector<double>* ST, std::vector<double>* SP, double* cfl_out, std::vector<double>* SX = nullptr) {
  const size_t N = o.N;
  const bool ext = use_pi && s.Pi && s.nB && SX;
  const int nf = use_pi ? (ext ? 16 : 14) : 4;
  const bool milne = (o.geometry == 0);
  const double tf = milne ? tau : 1.0;  // Q_T = tau*T_f^{tau mu}; Cartesian: factor 1
  PointTables pt;
  pt.P.resize(N); pt.cs2.resize(N); pt.T.resize(N); pt.c.resize(N);
  for (int m = 0; m < nf; ++m) { pt.Q[m].resize(N); pt.F[m].resize(N); }
  for (int m = 0; m < 4; ++m) ST[m].assign(N, 0.0);
  if (use_pi) for (int m = 0; m < 10; ++m) SP[m].assign(N, 0.0);
  if (ext) { SX[0].assign(N, 0.0); SX[1].assign(N, 0.0); }

  // step 1-2: EoS and conserved variables at every cell
#pragma omp parallel for if (N >= 2048)
  for (size_t c = 0; c < N; ++c) {
    double Tf[4][4], ut[4];
    eos_eval(o.eos, s.e[c], &pt.P[c], &pt.cs2[c], &pt.T[c]);
    frame_tensor(o, s, c, use_pi, pt.P[c], Tf, ut);
    for (int m = 0; m < 4; ++m) pt.Q[m][c] = tf * Tf[0][m];
    if (use_pi) for (int m = 0; m < 10; ++m) pt.Q[4 + m][c] = ut[0] * s.pi[m][c];
    if (ext) { pt.Q[14][c] = ut[0] * s.Pi[c]; pt.Q[15][c] = tf * s.nB[c] * ut[0]; }      // Eq.30; Eq.28 with A31
  }

  // steps 2-5: per axis, fluxes F_a, signal speed c_a, KT divergence (Eq.40); order x, y, eta (A22)
  for (int a = 0; a < 3; ++a) {
    double cflmax = 0.0;
    const double scale = (a == 2 && milne) ? 1.0 / (tau * o.d[2]) : 1.0 / o.d[a];
#pragma omp parallel for if (N >= 2048) reduction(max : cflmax)
    for (size_t c = 0; c < N; ++c) {
      double Tf[4][4], ut[4];
      frame_tensor(o, s, c, use_pi, pt.P[c], Tf, ut);
      for (int m = 0; m < 4; ++m) pt.F[m][c] = tf * Tf[a + 1][m];
      if (use_pi) for (int m = 0; m < 10; ++m) pt.F[4 + m][c] = ut[a + 1] * s.pi[m][c];
      if (ext) { pt.F[14][c] = ut[a + 1] * s.Pi[c]; pt.F[15][c] = tf * s.nB[c] * ut[a + 1]; }
      double g = ut[0];
      double v2 = (ut[1] * ut[1] + ut[2] * ut[2] + ut[3] * ut[3]) / (g * g);
      pt.c[c] = signal_speed(ut[a + 1] / g, v2, pt.cs2[c]);
      cflmax = std::max(cflmax, pt.c[c] * o.dtau * scale);
    }
    if (cfl_out) cfl_out[a] = cflmax;
#pragma omp parallel for if (N >= 2048)
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
        if (m < 4) ST[m][c] += div; else if (m < 14) SP[m - 4][c] += div; else SX[m - 14][c] += div;
      }
    }
  }

  // step 6-7: geometric source of T (Eq.31, sign A1), velocity gradients, IS source (Eq.33, A1, A2)
#pragma omp parallel for if (N >= 2048)
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
    double inv_taupi = T / (o.c_tau * o.eta_s * HBARC);     // tau_pi = 5 eta_v/(T s)
    double etav_over_taupi = (e + P) / o.c_tau;             // eta_v/tau_pi = (e+P)/5
    if (ext) {   // A29, A30: tau_Pi = tau_pi, zeta/tau_Pi = (zeta/s)/(eta_v/s) (e+P)/c_tau; S_N = 0 (Eq.32)
      double Pb = s.Pi[c];
      double src = -Pb * inv_taupi - (o.zeta_s / o.eta_s) * etav_over_taupi * theta_exp - Pb * theta_exp / 3.0;
      if (milne) src -= Pb * ut[0] / tau;
      SX[0][c] += src;
    }
    auto pic = [&](int m, int n) { return s.pi[PIDX[m][n]][c]; };
    // lambda_1 term (Eq.33): -(lambda_1/tau_pi) pi~^{<mu}_lambda pi~^{nu>lambda}, with the projector
    // of Eq.5 written out: X^{ab} = pi~^{a l} g~_{l k} pi~^{k b};  X^{<mn>} = Delta^{mn}_{ab} X^{ab},
    // Delta^{mn ab} = 1/2 (Delta^{ma} Delta^{nb} + Delta^{mb} Delta^{na}) - 1/3 Delta^{mn} Delta^{ab}.
    double PP[4][4] = {{0}};
    if (o.lambda1_hat != 0.0) {
      double X[4][4], Dl[4][4];   // Dl = Delta^{ab} = g~^{ab} - u~^a u~^b
      for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b) {
          X[a][b] = 0.0;
          for (int l = 0; l < 4; ++l) X[a][b] += pic(a, l) * GMET[l] * pic(l, b);
          Dl[a][b] = (a == b ? GMET[a] : 0.0) - ut[a] * ut[b];
        }
      for (int m = 0; m < 4; ++m)
        for (int n = 0; n < 4; ++n) {
          double acc = 0.0;
          for (int a = 0; a < 4; ++a)
            for (int b = 0; b < 4; ++b) {
              // indices of X lowered with g~: X_{ab} = g_aa g_bb X^{ab}
              double Xl = GMET[a] * GMET[b] * X[a][b];
              acc += (0.5 * (Dl[m][a] * Dl[n][b] + Dl[m][b] * Dl[n][a]) - Dl[m][n] * Dl[a][b] / 3.0) * Xl;
            }
          PP[m][n] = acc;
        }
    }
    for (int m = 0; m < 4; ++m)
      for (int n = m; n < 4; ++n) {
        // sigma~^{mu nu}: expansion of Eq.5
        double sig = GMET[m] * grad[m][n] + GMET[n] * grad[n][m] - ut[m] * Du[n] - ut[n] * Du[m]
                     - (2.0 / 3.0) * ((m == n ? GMET[m] : 0.0) - ut[m] * ut[n]) * theta_exp;
        double p = pic(m, n);
        double src = -p * inv_taupi + etav_over_taupi * sig - p * theta_exp / 3.0;
        if (o.lambda1_hat != 0.0) src -= (o.lambda1_hat / e) * inv_taupi * PP[m][n];
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
// Pib: bulk pressure carried through the root-find (A32; 0 without 8(f)-3).
void rootfind(Oracle& o, const double M[4], double* e_out, double u_out[3], long* nfloor, long* nclamp,
              double Pib = 0.0) {
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
    if (Pib != 0.0) { P += Pib; if (P < 0.0) { P = 0.0; cs2 = 0.0; } }   // A32: total pressure max(P + Pi, 0)
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
  if (Pib != 0.0) P = std::max(P + Pib, 0.0);
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

// Bulk limiter (A32): |Pi| <= xi P(e), so that P + Pi >= 0 for xi <= 1.
void limit_bulk(const Oracle& o, double e, double* Pib, long* nlimit) {
  if (!(o.xi > 0)) return;
  double P, cs2, T;
  eos_eval(o.eos, e, &P, &cs2, &T);
  double lim = o.xi * P;
  if (std::fabs(*Pib) > lim) { *Pib = std::copysign(lim, *Pib); ++*nlimit; }
}

State view(const std::vector<double>& e, const std::vector<double>* u, const std::vector<double>* pi,
           bool use_pi) {
  State s;
  s.e = e.data();
  for (int a = 0; a < 3; ++a) s.u[a] = u[a].data();
  for (int m = 0; m < 10; ++m) s.pi[m] = use_pi ? pi[m].data() : nullptr;
  return s;
}

// Q_T^mu = tf * T_f^{tau mu} of a state at one cell.
void conserved_T(const Oracle& o, const State& s, size_t c, bool use_pi, double tf, double QT[4]) {
  double P, cs2, T, Tf[4][4], ut[4];
  eos_eval(o.eos, s.e[c], &P, &cs2, &T);
  frame_tensor(o, s, c, use_pi, P, Tf, ut);
  for (int m = 0; m < 4; ++m) QT[m] = tf * Tf[0][m];
}

// Bootstrap of u^{-1} (A23; "ideal hydrodynamics is employed to estimate u*^1"):
// one ideal-fluid Euler predictor from (e, u~) with pi dropped gives u_id^1; u^{-1} = 2u^0 - u_id^1.
void bootstrap_history(Oracle& o) {
  const size_t N = o.N;
  const bool milne = (o.geometry == 0);
  State s = view(o.e, o.u, o.pi, false);
  std::vector<double> ST[4], SP[10];
  rhs(o, s, false, nullptr, o.tau0, ST, SP, nullptr);
  double tf0 = milne ? o.tau0 : 1.0, tf1 = milne ? o.tau0 + o.dtau : 1.0;
  long dummy1 = 0, dummy2 = 0;
#pragma omp parallel for if (N >= 2048) reduction(+ : dummy1, dummy2)
  for (size_t c = 0; c < N; ++c) {
    double QT[4], M[4], e1, u1[3];
    conserved_T(o, s, c, false, tf0, QT);
    for (int m = 0; m < 4; ++m) M[m] = (QT[m] + o.dtau * ST[m][c]) / tf1;
    rootfind(o, M, &e1, u1, &dummy1, &dummy2);
    for (int a = 0; a < 3; ++a) o.uprev[a][c] = 2.0 * o.u[a][c] - u1[a];
  }
}

// One full RK2 step n -> n+1  (Eq.49-54; readings A10-A12, A26).
void step_once(Oracle& o) {
  const size_t N = o.N;
  const bool milne = (o.geometry == 0);
  const bool visc = o.viscous();
  const double h = o.dtau;
  const double tau_n = o.tau0 + o.step * h, tau_1 = tau_n + h;
  const double tf_n = milne ? tau_n : 1.0, tf_1 = milne ? tau_1 : 1.0;

  // ---- stage 1 at tau_n -------------------------------------------------------------------
  std::vector<double> dtu[4], gstar(N);
  for (int m = 0; m < 4; ++m) dtu[m].resize(N);
#pragma omp parallel for if (N >= 2048)
  for (size_t c = 0; c < N; ++c) {
    double us[3], g2 = 1.0, gs2 = 1.0;
    for (int a = 0; a < 3; ++a) {
      us[a] = 2.0 * o.u[a][c] - o.uprev[a][c];          // u* = 2u^n - u^{n-1}
      g2 += o.u[a][c] * o.u[a][c];
      gs2 += us[a] * us[a];
    }
    gstar[c] = std::sqrt(gs2);                           // A11
    dtu[0][c] = (gstar[c] - std::sqrt(g2)) / h;          // A10
    for (int a = 0; a < 3; ++a) dtu[a + 1][c] = (us[a] - o.u[a][c]) / h;
  }
  const bool ext = visc && o.ext;
  State sn = view(o.e, o.u, o.pi, visc);
  if (ext) { sn.Pi = o.Pi.data(); sn.nB = o.nB.data(); }
  std::vector<double> ST[4], SP[10], SX[2];
  rhs(o, sn, visc, dtu, tau_n, ST, SP, o.cfl, ext ? SX : nullptr);

  std::vector<double> e1(N), u1[3], pi1[10], QTn[4];
  for (int a = 0; a < 3; ++a) u1[a].resize(N);
  for (int m = 0; m < 10; ++m) pi1[m].assign(N, 0.0);
  for (int m = 0; m < 4; ++m) QTn[m].resize(N);
  std::vector<double> Pi1, nb1, QNn;   // 8(f)-3: Pi', n' and Q_N^n
  if (ext) { Pi1.assign(N, 0.0); nb1.assign(N, 0.0); QNn.assign(N, 0.0); }
  long nfl = 0, ncl = 0, nli = 0, nbl = 0;   // event counters of this step (summed over the flat cell loops)
#pragma omp parallel for if (N >= 2048) reduction(+ : nfl, ncl, nli, nbl)
  for (size_t c = 0; c < N; ++c) {
    double QT[4], pp[10] = {0}, M[4], uu[3];
    conserved_T(o, sn, c, visc, tf_n, QT);
    for (int m = 0; m < 4; ++m) QTn[m][c] = QT[m];
    double gn = 1.0, Pb = 0.0;
    if (visc) {
      gn = std::sqrt(1.0 + o.u[0][c] * o.u[0][c] + o.u[1][c] * o.u[1][c] + o.u[2][c] * o.u[2][c]);
      for (int m = 0; m < 10; ++m) pp[m] = (gn * o.pi[m][c] + h * SP[m][c]) / gstar[c];   // Eq.49
    }
    if (ext) Pb = (gn * o.Pi[c] + h * SX[0][c]) / gstar[c];                                // Eq.48 like Eq.49
    for (int m = 0; m < 4; ++m) M[m] = (QT[m] + h * ST[m][c]) / tf_1 - pp[m];              // Eq.50-51
    rootfind(o, M, &e1[c], uu, &nfl, &ncl, Pb);
    if (visc) limit_pi(o, e1[c], pp, &nli);
    for (int a = 0; a < 3; ++a) u1[a][c] = uu[a];
    for (int m = 0; m < 10; ++m) pi1[m][c] = pp[m];
    if (ext) {
      limit_bulk(o, e1[c], &Pb, &nbl);
      Pi1[c] = Pb;
      QNn[c] = tf_n * o.nB[c] * gn;                                                        // Eq.46, A31
      double g1 = std::sqrt(1.0 + uu[0] * uu[0] + uu[1] * uu[1] + uu[2] * uu[2]);
      nb1[c] = (QNn[c] + h * SX[1][c]) / (tf_1 * g1);
    }
  }

  // ---- stage 2 at tau_{n+1} ---------------------------------------------------------------
#pragma omp parallel for if (N >= 2048)
  for (size_t c = 0; c < N; ++c) {
    double g2 = 1.0, g12 = 1.0;
    for (int a = 0; a < 3; ++a) { g2 += o.u[a][c] * o.u[a][c]; g12 += u1[a][c] * u1[a][c]; }
    dtu[0][c] = (std::sqrt(g12) - std::sqrt(g2)) / h;
    for (int a = 0; a < 3; ++a) dtu[a + 1][c] = (u1[a][c] - o.u[a][c]) / h;   // (u' - u^n)/h, A10
  }
  State s1 = view(e1, u1, pi1, visc);
  if (ext) { s1.Pi = Pi1.data(); s1.nB = nb1.data(); }
  std::vector<double> ST1[4], SP1[10], SX1[2];
  rhs(o, s1, visc, dtu, tau_1, ST1, SP1, nullptr, ext ? SX1 : nullptr);

  // Heun in Shu-Osher form (A26, default): Q^{n+1} = 1/2 [Q^n + Q(state') + h S_tot(state')], where
  // Q(state') is rebuilt from the stored stage-1 state (after floor / clamp / limiter).
  // heun_printed = 1: Eq.52-53 exactly as printed, Q^{n+1} = Q^n + h/2 (S_tot(n) + S_tot(')); the two agree to
  // rounding unless the floor, the v_max clamp or the pi limiter acted in stage 1.
  std::vector<double> pinew[10];
  for (int m = 0; m < 10; ++m) pinew[m].assign(N, 0.0);
  if (visc) {
#pragma omp parallel for if (N >= 2048)
    for (size_t c = 0; c < N; ++c) {
      double gn = std::sqrt(1.0 + o.u[0][c] * o.u[0][c] + o.u[1][c] * o.u[1][c] + o.u[2][c] * o.u[2][c]);
      double g1 = std::sqrt(1.0 + u1[0][c] * u1[0][c] + u1[1][c] * u1[1][c] + u1[2][c] * u1[2][c]);
      for (int m = 0; m < 10; ++m) {
        if (o.heun_printed)
          pinew[m][c] = (gn * o.pi[m][c] + 0.5 * h * (SP[m][c] + SP1[m][c])) / g1;             // Eq.52 as printed
        else
          pinew[m][c] = 0.5 * (gn * o.pi[m][c] + gstar[c] * pi1[m][c] + h * SP1[m][c]) / g1;   // Eq.52
      }
    }
    if (o.strict_eq53) {   // Eq.53 as printed: stage-2 T source evaluated with pi^{n+1} (A12)
      State s1b = view(e1, u1, pinew, true);
      std::vector<double> SPdummy[10];
      rhs(o, s1b, true, dtu, tau_1, ST1, SPdummy, nullptr);
    }
  }
#pragma omp parallel for if (N >= 2048) reduction(+ : nfl, ncl, nli, nbl)
  for (size_t c = 0; c < N; ++c) {
    double QT1[4], M[4], pp[10], en, uu[3];
    conserved_T(o, s1, c, visc, tf_1, QT1);
    for (int m = 0; m < 10; ++m) pp[m] = pinew[m][c];
    double Pb = 0.0, QNnew = 0.0;
    if (ext) {   // Heun for Pi and Q_N in the same bookkeeping as pi and Q_T (A26)
      double gn = std::sqrt(1.0 + o.u[0][c] * o.u[0][c] + o.u[1][c] * o.u[1][c] + o.u[2][c] * o.u[2][c]);
      double g1 = std::sqrt(1.0 + u1[0][c] * u1[0][c] + u1[1][c] * u1[1][c] + u1[2][c] * u1[2][c]);
      if (o.heun_printed) {
        Pb = (gn * o.Pi[c] + 0.5 * h * (SX[0][c] + SX1[0][c])) / g1;
        QNnew = QNn[c] + 0.5 * h * (SX[1][c] + SX1[1][c]);
      } else {
        Pb = 0.5 * (gn * o.Pi[c] + gstar[c] * Pi1[c] + h * SX1[0][c]) / g1;
        QNnew = 0.5 * (QNn[c] + tf_1 * nb1[c] * g1 + h * SX1[1][c]);
      }
    }
    for (int m = 0; m < 4; ++m) {
      if (o.heun_printed)
        M[m] = (QTn[m][c] + 0.5 * h * (ST[m][c] + ST1[m][c])) / tf_1 - pp[m];                // Eq.53-54 as printed
      else
        M[m] = 0.5 * (QTn[m][c] + QT1[m] + h * ST1[m][c]) / tf_1 - pp[m];                    // Eq.53-54
    }
    rootfind(o, M, &en, uu, &nfl, &ncl, Pb);
    if (visc) limit_pi(o, en, pp, &nli);
    for (int a = 0; a < 3; ++a) { o.uprev[a][c] = o.u[a][c]; o.u[a][c] = uu[a]; }
    o.e[c] = en;
    for (int m = 0; m < 10; ++m) o.pi[m][c] = pp[m];
    if (ext) {
      limit_bulk(o, en, &Pb, &nbl);
      o.Pi[c] = Pb;
      o.nB[c] = QNnew / (tf_1 * std::sqrt(1.0 + uu[0] * uu[0] + uu[1] * uu[1] + uu[2] * uu[2]));
    }
  }
  o.n_floor += nfl; o.n_clamp += ncl; o.n_limit += nli; o.n_bulk_limit += nbl;
  o.e_max_seen = *std::max_element(o.e.begin(), o.e.end());
  o.step += 1;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// C ABI (host pointers, fp64, unpadded component-major SoA [comp][nz][ny][nx], x fastest).
// ------------------------------------------------------------------------------------------
extern "C" {

void* oracle_create(int nx, int ny, int nz, double dx, double dy, double deta, const int* bc,
                    int geometry, double dtau, double tau0, int eos_kind, int eos_n, double e_min,
                    double e_max, const double* P, const double* T, double c_sb, double eta_over_s,
                    double minmod_theta, double e_floor, double pi_limit_xi, double v_max,
                    int strict_eq53) {
  if (nx < 1 || ny < 1 || nz < 1 || !(dtau > 0)) return nullptr;
  Oracle* o = new Oracle();
  o->nx = nx; o->ny = ny; o->nz = nz;
  o->d[0] = dx; o->d[1] = dy; o->d[2] = deta;
  for (int a = 0; a < 3; ++a) o->bc[a] = bc[a];
  o->geometry = geometry; o->dtau = dtau; o->tau0 = tau0; o->eta_s = eta_over_s;
  o->eos.kind = eos_kind; o->eos.n = eos_n; o->eos.e_min = e_min; o->eos.e_max = e_max;
  o->eos.c_sb = c_sb;
  if (eos_kind == 1) { o->eos.P.assign(P, P + eos_n); o->eos.T.assign(T, T + eos_n); }
  o->theta = minmod_theta; o->e_floor = e_floor; o->xi = pi_limit_xi; o->v_max = v_max;
  o->strict_eq53 = strict_eq53;
  o->N = size_t(nx) * ny * nz;
  o->e.assign(o->N, 0.0);
  for (int a = 0; a < 3; ++a) { o->u[a].assign(o->N, 0.0); o->uprev[a].assign(o->N, 0.0); }
  for (int m = 0; m < 10; ++m) o->pi[m].assign(o->N, 0.0);
  return o;
}

void oracle_destroy(void* h) { delete static_cast<Oracle*>(h); }

// T: T_f^{tau mu} [4][N] (no extra factor tau); pi: pi~ [10][N] or NULL.  8(f)-3 (ext = 1): Pi [N] and nb [N] (NULL = 0);
// T is then the full tensor, including the bulk pressure (A28), and the root-find carries Pi (A32).
int oracle_load_ext(void* h, const double* T, const double* pi, const double* Pi, const double* nb) {
  Oracle& o = *static_cast<Oracle*>(h);
  const size_t N = o.N;
  const bool ext = o.ext && o.viscous();
  if (ext) { o.Pi.assign(N, 0.0); o.nB.assign(N, 0.0); }
  long nfl = 0, ncl = 0;
#pragma omp parallel for if (N >= 2048) reduction(+ : nfl, ncl)
  for (size_t c = 0; c < N; ++c) {
    double M[4], uu[3];
    for (int m = 0; m < 10; ++m) o.pi[m][c] = (pi && o.viscous()) ? pi[m * N + c] : 0.0;
    for (int m = 0; m < 4; ++m) M[m] = T[m * N + c] - o.pi[m][c];
    if (ext) { o.Pi[c] = Pi ? Pi[c] : 0.0; o.nB[c] = nb ? nb[c] : 0.0; }
    rootfind(o, M, &o.e[c], uu, &nfl, &ncl, ext ? o.Pi[c] : 0.0);
    for (int a = 0; a < 3; ++a) o.u[a][c] = uu[a];
  }
  o.n_floor += nfl; o.n_clamp += ncl;
  o.step = 0;
  bootstrap_history(o);
  o.e_max_seen = *std::max_element(o.e.begin(), o.e.end());
  o.loaded = true;
  return 0;
}

int oracle_load(void* h, const double* T, const double* pi) { return oracle_load_ext(h, T, pi, nullptr, nullptr); }

// 8(f)-3: bulk pressure Pi [N] and net-baryon density n [N] of the current state; either may be NULL.
int oracle_read_ext(void* h, double* Pi, double* nb) {
  Oracle& o = *static_cast<Oracle*>(h);
  const bool ext = o.ext && o.viscous();
  for (size_t c = 0; c < o.N; ++c) {
    if (Pi) Pi[c] = ext ? o.Pi[c] : 0.0;
    if (nb) nb[c] = ext ? o.nB[c] : 0.0;
  }
  return 0;
}

// Overwrite the history u~^i_{n-1} [3][N] (analytic tests that know the exact earlier level).
int oracle_set_history(void* h, const double* uprev) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int a = 0; a < 3; ++a) std::copy(uprev + a * o.N, uprev + (a + 1) * o.N, o.uprev[a].begin());
  return 0;
}

int oracle_step(void* h, int n) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (!o.loaded) return -4;
  for (int s = 0; s < n; ++s) step_once(o);
  return 0;
}

// e [N], u~^mu [4][N], pi~ [10][N]; any may be NULL.
int oracle_read(void* h, double* e, double* u, double* pi) {
  Oracle& o = *static_cast<Oracle*>(h);
  const size_t N = o.N;
  for (size_t c = 0; c < N; ++c) {
    if (e) e[c] = o.e[c];
    if (u) {
      u[c] = std::sqrt(1.0 + o.u[0][c] * o.u[0][c] + o.u[1][c] * o.u[1][c] + o.u[2][c] * o.u[2][c]);
      for (int a = 0; a < 3; ++a) u[(a + 1) * N + c] = o.u[a][c];
    }
    if (pi) for (int m = 0; m < 10; ++m) pi[m * N + c] = o.pi[m][c];
  }
  return 0;
}

// T_f^{tau mu} [4][N] of the current state.
int oracle_read_T(void* h, double* T) {
  Oracle& o = *static_cast<Oracle*>(h);
  State s = view(o.e, o.u, o.pi, o.viscous());
  if (o.ext && o.viscous() && o.Pi.size() == o.N) s.Pi = o.Pi.data();      // 8(f)-3: the full tensor (A28)
  for (size_t c = 0; c < o.N; ++c) {
    double QT[4];
    conserved_T(o, s, c, o.viscous(), 1.0, QT);
    for (int m = 0; m < 4; ++m) T[m * o.N + c] = QT[m];
  }
  return 0;
}

int oracle_read_history(void* h, double* uprev) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int a = 0; a < 3; ++a) std::copy(o.uprev[a].begin(), o.uprev[a].end(), uprev + a * o.N);
  return 0;
}

// diag[0]=tau, [1]=step, [2..4]=CFL per axis (last stage 1), [5]=e_max, [6]=floored, [7]=clamped,
// [8]=pi-limited (cumulative counts).
int oracle_diag(void* h, double* diag) {
  Oracle& o = *static_cast<Oracle*>(h);
  diag[0] = o.tau0 + o.step * o.dtau; diag[1] = o.step;
  for (int a = 0; a < 3; ++a) diag[2 + a] = o.cfl[a];
  diag[5] = o.e_max_seen; diag[6] = double(o.n_floor); diag[7] = double(o.n_clamp);
  diag[8] = double(o.n_limit);
  return 0;
}

// RHS operator on the current state with a caller-supplied d_tau u~ [4][N] (test hook for the
// brute-force and PDE-residual pins).  ST [4][N], SP [10][N].
int oracle_rhs(void* h, const double* dtu, double tau, double* ST, double* SP) {
  Oracle& o = *static_cast<Oracle*>(h);
  const size_t N = o.N;
  std::vector<double> d[4], st[4], sp[10];
  for (int m = 0; m < 4; ++m) d[m].assign(dtu + m * N, dtu + (m + 1) * N);
  State s = view(o.e, o.u, o.pi, o.viscous());
  rhs(o, s, o.viscous(), d, tau, st, sp, nullptr);
  for (int m = 0; m < 4; ++m) std::copy(st[m].begin(), st[m].end(), ST + m * N);
  if (o.viscous() && SP) for (int m = 0; m < 10; ++m) std::copy(sp[m].begin(), sp[m].end(), SP + m * N);
  return 0;
}

// Directly set the state (e [N], u~^i [3][N], pi~ [10][N] or NULL) without a root-find.
int oracle_set_state(void* h, const double* e, const double* u, const double* pi) {
  Oracle& o = *static_cast<Oracle*>(h);
  const size_t N = o.N;
  std::copy(e, e + N, o.e.begin());
  for (int a = 0; a < 3; ++a) std::copy(u + a * N, u + (a + 1) * N, o.u[a].begin());
  for (int m = 0; m < 10; ++m)
    for (size_t c = 0; c < N; ++c) o.pi[m][c] = (pi && o.viscous()) ? pi[m * N + c] : 0.0;
  o.uprev[0] = o.u[0]; o.uprev[1] = o.u[1]; o.uprev[2] = o.u[2];
  if (o.ext && o.viscous()) { o.Pi.assign(N, 0.0); o.nB.assign(N, 0.0); }
  o.step = 0; o.loaded = true;
  return 0;
}

// 8(f)-3: set Pi [N] and n [N] of the current state directly (after oracle_set_state); NULL leaves a field as it is.
int oracle_set_ext(void* h, const double* Pi, const double* nb) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (!(o.ext && o.viscous())) return -1;
  if (o.Pi.size() != o.N) { o.Pi.assign(o.N, 0.0); o.nB.assign(o.N, 0.0); }
  if (Pi) std::copy(Pi, Pi + o.N, o.Pi.begin());
  if (nb) std::copy(nb, nb + o.N, o.nB.begin());
  return 0;
}

void oracle_eos(void* h, double e, double* out3) {
  Oracle& o = *static_cast<Oracle*>(h);
  eos_eval(o.eos, e, &out3[0], &out3[1], &out3[2]);
}

// Test hook: the pi limiter (A14) on one cell; pi10 is scaled in place, returns 1 when it acted.
int oracle_limit_pi(void* h, double e, double* pi10) {
  Oracle& o = *static_cast<Oracle*>(h);
  long n = 0;
  limit_pi(o, e, pi10, &n);
  return int(n);
}

// Options that are not part of oracle_create's argument list.  key 0: heun_printed (A26; 0 default, 1 = Eq.52-53
// as printed); key 1: lambda1_hat; key 2: c_tau; keys 3, 4: SURVEY 8(f)-3.  Returns 0, or -1 for an
// unknown key / bad value.
int oracle_set_option(void* h, int key, double value) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (key == 0) { o.heun_printed = value != 0.0 ? 1 : 0; return 0; }
  if (key == 1) { o.lambda1_hat = value; return 0; }
  if (key == 2) { if (!(value > 0.0)) return -1; o.c_tau = value; return 0; }
  // key 3: evolve Pi and n (8(f)-3; viscous runs without strict_eq53 only); key 4: zeta/s >= 0 (A30)
  if (key == 3) { if (value != 0.0 && (!o.viscous() || o.strict_eq53)) return -1; o.ext = value != 0.0 ? 1 : 0; return 0; }
  if (key == 4) { if (!(value >= 0.0)) return -1; o.zeta_s = value; return 0; }
  return -1;
}

void oracle_rootfind(void* h, const double* M4, double* out4) {
  Oracle& o = *static_cast<Oracle*>(h);
  long a = 0, b = 0;
  rootfind(o, M4, &out4[0], &out4[1], &a, &b);
}

}  // extern "C"
