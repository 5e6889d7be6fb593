// ============================================================================
// grpic_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct FP64 CPU restatement of the GRPIC hot path of
// arxiv 2503.04558 ("Introducing APERTURE: a GPU-based GRPIC framework"), written
// step by step from /root/reference/PAPER.md in the paper's order and notation.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may load this library.  It shares no code, header, table or
// helper with paper_2503_04558_b200/csrc (the CUDA product path) and neither
// includes the other.
//
// What pins each function (tests/test_oracle_*.py, -m "not gpu"):
//   orc_metric            inverse identity, det gamma, finite-difference derivatives
//   orc_gauss_legendre    numpy.polynomial.legendre.leggauss
//   orc_areas             scipy.integrate.quad; a=0 closed forms
//   orc_geodesic*         u_phi exact, E=-u_t ~ dt^2, Table 1 energies/periods, ISCO Omega
//   orc_boris             norm conservation, Eq.16 residual, flat-space gyration
//   orc_vay               E x B drift held exactly, |u| exact in pure B, agrees with Boris to O(dt^2)
//   orc_push (+Wald)      Eq.24 energy and canonical L_phi conservation
//   orc_deposit           discrete continuity Eq.21 to round-off; whole-row brute force
//   orc_circulation/field div B exactly preserved; div D - rho preserved; Wald/monopole
//                         stationarity ~ Delta^2; Heun limit / order in dt
//   orc_sort/orc_compact  = std::stable_sort / order-preserving filter (library definition)
//   orc_ks_to_bl          Boyer-Lindquist normalisation g_BL^{mu nu} u_mu u_nu = -eps with the textbook BL
//                         inverse metric; (A7) differentiated against (A6); u_i = 0 gives Gamma = 1
//   orc_sort_interleaved  numpy lexsort of the defining tuple; hand-built example; B = 1 reduces to orc_sort
//   shape option 3        cubic B-spline: partition of unity, moments, C2 knots; continuity to
//                         round-off with the spline in rho and fluxes; exact gather of linear fields
//   orc_philox4x32_10     the published known-answer vectors (tests/golden/philox4x32_10.txt)
//   orc_pair_production   FIDO momentum / energy conservation, eps_ph, threshold, Eq.26 fraction,
//                         append order; recoil and split prescriptions are readings P1-P4
//   PARITY UNPINNED (paper silent; reading listed in DESIGN.md): field gather at
//   staggered positions (G11/G12), damping profile (G14), current filter (S10),
//   log-r basis choice (G8).
//
// Array layout of THIS file (independent of the CUDA library's pitched layout):
// every grid array is [nth+1+2G][nr+1+2G] doubles, r fastest, G = ng;
// logical index (i,j), i in [-G,nr+G], j in [-G,nth+G] -> (j+G)*NRP + (i+G).
// Staggering (Fig.1, B8-B11 :480-517), index (i,j) means position
//   D^r,J^r,E_r,B^th,H_th : (i+1/2, j)      D^th,J^th,E_th,B^r,H_r : (i, j+1/2)
//   D^ph,J^ph,E_ph,rho    : (i, j)          B^ph,H_ph              : (i+1/2, j+1/2)
// xi = ln r, xi_i = xi_in + i*dxi, theta_j = j*dth.
// ============================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

struct orc_params {
  double a, M;
  int32_t nr, nth, ng;
  double xi_in, xi_out, dphi;
  int32_t geo_iters, field_iters;
  double beta_impl;
  int32_t damp_cells;
  double damp_coef;
};

}  // extern "C"

namespace {

struct Grid {
  int nr, nth, G, NRP, NTHP;
  double xi_in, dxi, dth, dphi, a, M;
  explicit Grid(const orc_params& p)
      : nr(p.nr), nth(p.nth), G(p.ng), NRP(p.nr + 1 + 2 * p.ng), NTHP(p.nth + 1 + 2 * p.ng),
        xi_in(p.xi_in), dxi((p.xi_out - p.xi_in) / p.nr), dth(M_PI / p.nth), dphi(p.dphi),
        a(p.a), M(p.M) {}
  size_t idx(int i, int j) const { return (size_t)(j + G) * NRP + (i + G); }
  size_t size() const { return (size_t)NRP * NTHP; }
  double xi(double i) const { return xi_in + i * dxi; }
  double r(double i) const { return std::exp(xi(i)); }
  double th(double j) const { return j * dth; }
};

// ---------------------------------------------------------------------------
// Kerr-Schild 3+1 metric, Appendix A, M restored
// (z = 2Mr/rho^2, Delta = r^2 + a^2 - 2Mr).
// ---------------------------------------------------------------------------
struct Metric {
  double alpha, beta_r;                   // (A5)
  double g_rr, g_thth, g_phph, g_rph;     // gamma_ij (A2)
  double gu_rr, gu_thth, gu_phph, gu_rph; // gamma^ij (A4)
  double sqrtg;                           // sqrt(det gamma_ij)
  // derivatives w.r.t. r and theta of alpha, beta^r and gamma^ij
  double dr_alpha, dth_alpha, dr_beta, dth_beta;
  double dr_gu_rr, dth_gu_rr, dr_gu_thth, dth_gu_thth, dr_gu_phph, dth_gu_phph, dr_gu_rph,
      dth_gu_rph;
};

Metric metric(double a, double M, double r, double th) {
  Metric m;
  const double s = std::sin(th), c = std::cos(th);
  const double s2 = s * s, c2 = c * c;
  const double rho2 = r * r + a * a * c2;            // (A3)
  const double z = 2.0 * M * r / rho2;               // (A3)
  const double Delta = r * r + a * a - 2.0 * M * r;  // (A3)
  const double Sigma = (r * r + a * a) * (r * r + a * a) - a * a * Delta * s2;  // (A3)
  m.alpha = 1.0 / std::sqrt(1.0 + z);                // (A5)
  m.beta_r = z / (1.0 + z);                          // (A5)
  m.g_rr = 1.0 + z;                                  // (A2)
  m.g_thth = rho2;
  m.g_phph = Sigma * s2 / rho2;
  m.g_rph = -a * s2 * (1.0 + z);
  m.gu_rr = (a * a + r * r) / rho2 - 2.0 * M * r / (rho2 + 2.0 * M * r);  // (A4)
  m.gu_thth = 1.0 / rho2;
  m.gu_phph = 1.0 / (rho2 * s2);
  m.gu_rph = a / rho2;
  m.sqrtg = rho2 * s * std::sqrt(1.0 + z);  // sqrt(det gamma); pinned by det identity test
  // ---- derivatives (own derivation; pinned by finite differences) ----
  const double drho2_dr = 2.0 * r, drho2_dth = -2.0 * a * a * s * c;
  const double dz_dr = 2.0 * M / rho2 - 2.0 * M * r * drho2_dr / (rho2 * rho2);
  const double dz_dth = -2.0 * M * r * drho2_dth / (rho2 * rho2);
  // alpha = (1+z)^(-1/2)
  m.dr_alpha = -0.5 * std::pow(1.0 + z, -1.5) * dz_dr;
  m.dth_alpha = -0.5 * std::pow(1.0 + z, -1.5) * dz_dth;
  // beta^r = z/(1+z)  ->  d = dz/(1+z)^2
  m.dr_beta = dz_dr / ((1.0 + z) * (1.0 + z));
  m.dth_beta = dz_dth / ((1.0 + z) * (1.0 + z));
  // gamma^rr = (r^2+a^2)/rho2 - z/(1+z)
  m.dr_gu_rr = 2.0 * r / rho2 - (r * r + a * a) * drho2_dr / (rho2 * rho2) - m.dr_beta;
  m.dth_gu_rr = -(r * r + a * a) * drho2_dth / (rho2 * rho2) - m.dth_beta;
  // gamma^thth = 1/rho2
  m.dr_gu_thth = -drho2_dr / (rho2 * rho2);
  m.dth_gu_thth = -drho2_dth / (rho2 * rho2);
  // gamma^phph = 1/(rho2 s^2)
  m.dr_gu_phph = -drho2_dr / (rho2 * rho2 * s2);
  m.dth_gu_phph = -drho2_dth / (rho2 * rho2 * s2) - 2.0 * c / (rho2 * s2 * s);
  // gamma^rph = a/rho2
  m.dr_gu_rph = -a * drho2_dr / (rho2 * rho2);
  m.dth_gu_rph = -a * drho2_dth / (rho2 * rho2);
  return m;
}

// ---------------------------------------------------------------------------
// 10-point Gauss-Legendre rule on [-1,1], nodes by Newton on P_n.
// ---------------------------------------------------------------------------
void gauss_legendre(int n, double* x, double* w) {
  for (int k = 0; k < n; ++k) {
    double t = std::cos(M_PI * (k + 0.75) / (n + 0.5));
    double dp = 0.0;
    for (int it = 0; it < 100; ++it) {
      double p0 = 1.0, p1 = t;
      for (int l = 2; l <= n; ++l) {
        double p2 = ((2.0 * l - 1.0) * t * p1 - (l - 1.0) * p0) / l;
        p0 = p1;
        p1 = p2;
      }
      dp = n * (t * p1 - p0) / (t * t - 1.0);
      double dt = p1 / dp;
      t -= dt;
      if (std::fabs(dt) < 1e-16) break;
    }
    // re-evaluate derivative at the converged node
    double p0 = 1.0, p1 = t;
    for (int l = 2; l <= n; ++l) {
      double p2 = ((2.0 * l - 1.0) * t * p1 - (l - 1.0) * p0) / l;
      p0 = p1;
      p1 = p2;
    }
    dp = n * (t * p1 - p0) / (t * t - 1.0);
    x[k] = t;
    w[k] = 2.0 / ((1.0 - t * t) * dp * dp);
  }
}

struct GL10 {
  double x[10], w[10];
  GL10() { gauss_legendre(10, x, w); }
};

// integral of sqrt(gamma) over theta in [t0,t1] at fixed r
double int_th(const Grid& g, const GL10& q, double r, double t0, double t1) {
  if (t1 <= t0) return 0.0;
  double sum = 0.0;
  for (int k = 0; k < 10; ++k) {
    double t = 0.5 * (t0 + t1) + 0.5 * (t1 - t0) * q.x[k];
    sum += q.w[k] * metric(g.a, g.M, r, t).sqrtg;
  }
  return 0.5 * (t1 - t0) * sum;
}
// integral of sqrt(gamma) dr = sqrt(gamma) r dxi over xi in [x0,x1] at fixed theta
double int_xi(const Grid& g, const GL10& q, double th, double x0, double x1) {
  double sum = 0.0;
  for (int k = 0; k < 10; ++k) {
    double x = 0.5 * (x0 + x1) + 0.5 * (x1 - x0) * q.x[k];
    double r = std::exp(x);
    sum += q.w[k] * metric(g.a, g.M, r, th).sqrtg * r;
  }
  return 0.5 * (x1 - x0) * sum;
}
double int_xi_th(const Grid& g, const GL10& q, double x0, double x1, double t0, double t1) {
  if (t1 <= t0) return 0.0;
  double sum = 0.0;
  for (int k = 0; k < 10; ++k) {
    double x = 0.5 * (x0 + x1) + 0.5 * (x1 - x0) * q.x[k];
    double r = std::exp(x);
    sum += q.w[k] * r * int_th(g, q, r, t0, t1);
  }
  return 0.5 * (x1 - x0) * sum;
}
double clip(double t) { return std::min(std::max(t, 0.0), M_PI); }

// Area elements, Eq.(8), D- and B-staggered sets.
struct Areas {
  std::vector<double> ADr, ADth, ADph, ABr, ABth, ABph;
};
void compute_areas(const Grid& g, double* ADr, double* ADth, double* ADph, double* ABr,
                   double* ABth, double* ABph) {
  GL10 q;
  for (size_t k = 0; k < g.size(); ++k) ADr[k] = ADth[k] = ADph[k] = ABr[k] = ABth[k] = ABph[k] = 0.0;
  // rows are independent (every iteration writes only its own node): the OpenMP loop over rows is
  // bit-identical to the serial one (tests/test_oracle_grid.py::test_field_step_threads_bit_identical)
#pragma omp parallel for schedule(static)
  for (int j = 0; j <= g.nth; ++j)
    for (int i = -g.G; i <= g.nr + g.G; ++i) {
      const size_t k = g.idx(i, j);
      const double tlo = clip(g.th(j - 0.5)), thi = clip(g.th(j + 0.5));
      // A^D_r at (i+1/2, j): dual face in theta (clipped at the axes)
      ADr[k] = g.dphi * int_th(g, q, g.r(i + 0.5), tlo, thi);
      // A^D_phi at (i,j): dual cell
      ADph[k] = int_xi_th(g, q, g.xi(i - 0.5), g.xi(i + 0.5), tlo, thi);
      // A^B_theta at (i+1/2, j): primal edge in r (vanishes on the axes)
      ABth[k] = g.dphi * int_xi(g, q, g.th(j), g.xi(i), g.xi(i + 1));
      if (j < g.nth) {
        // A^D_theta at (i, j+1/2): dual edge in r
        ADth[k] = g.dphi * int_xi(g, q, g.th(j + 0.5), g.xi(i - 0.5), g.xi(i + 0.5));
        // A^B_r at (i, j+1/2): primal face in theta
        ABr[k] = g.dphi * int_th(g, q, g.r(i), g.th(j), g.th(j + 1));
        // A^B_phi at (i+1/2, j+1/2): primal cell
        ABph[k] = int_xi_th(g, q, g.xi(i), g.xi(i + 1), g.th(j), g.th(j + 1));
      }
    }
}

// ---------------------------------------------------------------------------
// Field gather, first order.  Reading G11/G12:
// bilinear in (xi,theta) index space from each component's own staggered
// lattice; theta-ghost values by parity about the axis (r,phi components even,
// theta components odd); radial guard values are read as stored.
// ---------------------------------------------------------------------------
struct Stag {
  double sr, sth;  // stagger offsets (0 or 1/2)
  int parity;      // +1 even, -1 odd under theta -> -theta
};
const Stag ST_Dr{0.5, 0.0, +1}, ST_Dth{0.0, 0.5, -1}, ST_Dph{0.0, 0.0, +1};
const Stag ST_Br{0.0, 0.5, +1}, ST_Bth{0.5, 0.0, -1}, ST_Bph{0.5, 0.5, +1};

double fetch(const Grid& g, const double* F, const Stag& st, int i, int j) {
  double sign = 1.0;
  if (st.sth == 0.0) {  // node-located in theta: rows 0..nth
    if (j < 0) { j = -j; sign = st.parity; }
    if (j > g.nth) { j = 2 * g.nth - j; sign = st.parity; }
  } else {  // half-staggered in theta: rows 0..nth-1 at (j+1/2)
    if (j < 0) { j = -1 - j; sign = st.parity; }
    if (j > g.nth - 1) { j = 2 * g.nth - 1 - j; sign = st.parity; }
  }
  return sign * F[g.idx(i, j)];
}

int g_shape_order = 1;   // shape option, see shape() below
double shape(double x);
double gather1(const Grid& g, const double* F, const Stag& st, double fx, double fy) {
  const double gx = fx - st.sr, gy = fy - st.sth;
  const int i0 = (int)std::floor(gx), j0 = (int)std::floor(gy);
  if (g_shape_order == 3) {                          // sum over the 4 x 4 nodes of the spline's support
    double acc = 0.0;
    for (int j = j0 - 1; j <= j0 + 2; ++j)
      for (int i = i0 - 1; i <= i0 + 2; ++i) acc += shape(gx - i) * shape(gy - j) * fetch(g, F, st, i, j);
    return acc;
  }
  const double wx = gx - i0, wy = gy - j0;
  return (1.0 - wy) * ((1.0 - wx) * fetch(g, F, st, i0, j0) + wx * fetch(g, F, st, i0 + 1, j0)) +
         wy * ((1.0 - wx) * fetch(g, F, st, i0, j0 + 1) + wx * fetch(g, F, st, i0 + 1, j0 + 1));
}

// ---------------------------------------------------------------------------
// Generalised Boris push, full dt, Eq.(16)-(19) PAPER.md:176-200.
// sgn = q/m = +-1.  D[3], B[3] contravariant (r,theta,phi); u covariant.
// ---------------------------------------------------------------------------
void lower(const Metric& m, const double v[3], double out[3]) {
  out[0] = m.g_rr * v[0] + m.g_rph * v[2];
  out[1] = m.g_thth * v[1];
  out[2] = m.g_rph * v[0] + m.g_phph * v[2];
}
void raise(const Metric& m, const double v[3], double out[3]) {
  out[0] = m.gu_rr * v[0] + m.gu_rph * v[2];
  out[1] = m.gu_thth * v[1];
  out[2] = m.gu_rph * v[0] + m.gu_phph * v[2];
}
// (a x b)_i = sqrt(gamma) eps_ijk a^j b^k   (covariant result from contravariant inputs)
void cross_lo(const Metric& m, const double a[3], const double b[3], double out[3]) {
  out[0] = m.sqrtg * (a[1] * b[2] - a[2] * b[1]);
  out[1] = m.sqrtg * (a[2] * b[0] - a[0] * b[2]);
  out[2] = m.sqrtg * (a[0] * b[1] - a[1] * b[0]);
}
double norm_up(const Metric& m, const double u[3]) {  // gamma^ij u_i u_j
  return m.gu_rr * u[0] * u[0] + m.gu_thth * u[1] * u[1] + m.gu_phph * u[2] * u[2] +
         2.0 * m.gu_rph * u[0] * u[2];
}

void boris(const Metric& m, const double u[3], const double D[3], const double B[3], double sgn,
           double dt, double uout[3]) {
  double Dlo[3];
  lower(m, D, Dlo);
  double um[3];  // u^-  (17)
  for (int k = 0; k < 3; ++k) um[k] = u[k] + sgn * (m.alpha * dt / 2.0) * Dlo[k];
  const double u0bar = std::sqrt(1.0 + norm_up(m, um)) / m.alpha;  // (18)
  double t[3];                                                      // (17)
  for (int k = 0; k < 3; ++k) t[k] = sgn * B[k] * dt / (2.0 * u0bar);
  double um_up[3], cr[3], ut[3];
  raise(m, um, um_up);
  cross_lo(m, um_up, t, cr);
  for (int k = 0; k < 3; ++k) ut[k] = um[k] + cr[k];  // u~ (19)
  double tlo[3];
  lower(m, t, tlo);
  const double t2 = t[0] * tlo[0] + t[1] * tlo[1] + t[2] * tlo[2];
  double s[3];
  for (int k = 0; k < 3; ++k) s[k] = 2.0 * t[k] / (1.0 + t2);  // (19)
  double ut_up[3], up[3];
  raise(m, ut, ut_up);
  cross_lo(m, ut_up, s, cr);
  for (int k = 0; k < 3; ++k) up[k] = um[k] + cr[k];  // u^+ (19)
  for (int k = 0; k < 3; ++k) uout[k] = up[k] + sgn * (m.alpha * dt / 2.0) * Dlo[k];  // (17)
}

// Vay pusher in the FIDO frame ("a transformation to the FIDO frame and ... the
// Vay momentum update there (Vay 2008)").  Readings V1-V3: orthonormal triad
//   e_(1) = sqrt(gamma^rr) (d_r - (gamma_rphi/gamma_phiphi) d_phi),  e_(2) = d_theta/sqrt(gamma_thth),
//   e_(3) = d_phi/sqrt(gamma_phiphi)   (right-handed: sqrt(gamma) eps_ijk e1^i e2^j e3^k = 1);
// FIDO proper time of the step alpha*dt; D^i, B^i are the fields the FIDO measures.  Vay (2008):
//   u' = u + h (E + v x B / 2),  v = u/Gamma,  h = (q/m) alpha dt,  tau = (h/2) B,  u* = u'.tau,
//   sigma = 1 + u'^2 - tau^2,  Gamma1^2 = (sigma + sqrt(sigma^2 + 4 (tau^2 + u*^2)))/2,
//   t = tau/Gamma1,  u1 = (u' + (u'.t) t + u' x t)/(1 + t^2).
void vay(const Metric& m, const double u[3], const double D[3], const double B[3], double sgn, double dt,
         double uout[3]) {
  const double sgrr = std::sqrt(m.gu_rr), sth = std::sqrt(m.g_thth), sph = std::sqrt(m.g_phph);
  const double k = m.g_rph / m.g_phph;
  auto vec_hat = [&](const double V[3], double out[3]) {          // contravariant -> orthonormal
    out[0] = V[0] / sgrr;
    out[1] = sth * V[1];
    out[2] = (m.g_rph * V[0] + m.g_phph * V[2]) / sph;
  };
  const double uh[3] = {sgrr * (u[0] - k * u[2]), u[1] / sth, u[2] / sph};   // covariant -> orthonormal
  double E[3], Bh[3];
  vec_hat(D, E);
  vec_hat(B, Bh);
  const double h = sgn * m.alpha * dt;
  const double G0 = std::sqrt(1.0 + uh[0] * uh[0] + uh[1] * uh[1] + uh[2] * uh[2]);
  const double v[3] = {uh[0] / G0, uh[1] / G0, uh[2] / G0};
  double up[3];
  up[0] = uh[0] + h * (E[0] + 0.5 * (v[1] * Bh[2] - v[2] * Bh[1]));
  up[1] = uh[1] + h * (E[1] + 0.5 * (v[2] * Bh[0] - v[0] * Bh[2]));
  up[2] = uh[2] + h * (E[2] + 0.5 * (v[0] * Bh[1] - v[1] * Bh[0]));
  const double tau[3] = {0.5 * h * Bh[0], 0.5 * h * Bh[1], 0.5 * h * Bh[2]};
  const double tau2 = tau[0] * tau[0] + tau[1] * tau[1] + tau[2] * tau[2];
  const double ustar = up[0] * tau[0] + up[1] * tau[1] + up[2] * tau[2];
  const double sigma = 1.0 + up[0] * up[0] + up[1] * up[1] + up[2] * up[2] - tau2;
  const double G1 = std::sqrt(0.5 * (sigma + std::sqrt(sigma * sigma + 4.0 * (tau2 + ustar * ustar))));
  const double t[3] = {tau[0] / G1, tau[1] / G1, tau[2] / G1};
  const double t2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
  const double udt = up[0] * t[0] + up[1] * t[1] + up[2] * t[2];
  const double sc = 1.0 / (1.0 + t2);
  const double u1[3] = {sc * (up[0] + udt * t[0] + (up[1] * t[2] - up[2] * t[1])),
                        sc * (up[1] + udt * t[1] + (up[2] * t[0] - up[0] * t[2])),
                        sc * (up[2] + udt * t[2] + (up[0] * t[1] - up[1] * t[0]))};
  uout[0] = u1[0] / sgrr + u1[2] * m.g_rph / sph;                 // orthonormal -> covariant
  uout[1] = sth * u1[1];
  uout[2] = sph * u1[2];
}
int g_pusher = 0;   // momentum update of orc_push: 0 = generalised Boris (default), 1 = Vay in the FIDO frame

// ---------------------------------------------------------------------------
// Geodesic right-hand sides X^i, U_i of Eq.(12) without F_i,
// y = (r, theta, phi, u_r, u_theta, u_phi); eps = 1 massive, 0 photon (:153).
// ---------------------------------------------------------------------------
void geodesic_rhs(double a, double M, const double y[6], double eps, double f[6]) {
  const Metric m = metric(a, M, y[0], y[1]);
  const double* u = y + 3;
  const double u0 = std::sqrt(eps + norm_up(m, u)) / m.alpha;
  f[0] = (m.gu_rr * u[0] + m.gu_rph * u[2]) / u0 - m.beta_r;
  f[1] = m.gu_thth * u[1] / u0;
  f[2] = (m.gu_phph * u[2] + m.gu_rph * u[0]) / u0;
  const double dr_quad = m.dr_gu_rr * u[0] * u[0] + m.dr_gu_thth * u[1] * u[1] +
                         m.dr_gu_phph * u[2] * u[2] + 2.0 * m.dr_gu_rph * u[0] * u[2];
  const double dth_quad = m.dth_gu_rr * u[0] * u[0] + m.dth_gu_thth * u[1] * u[1] +
                          m.dth_gu_phph * u[2] * u[2] + 2.0 * m.dth_gu_rph * u[0] * u[2];
  f[3] = -m.alpha * u0 * m.dr_alpha + u[0] * m.dr_beta - dr_quad / (2.0 * u0);
  f[4] = -m.alpha * u0 * m.dth_alpha + u[0] * m.dth_beta - dth_quad / (2.0 * u0);
  f[5] = 0.0;
}

// Predictor (14) + K trapezoidal correctors (15); each corrector
// re-evaluates the RHS at the previous iterate (reading G10).
void geodesic(double a, double M, int K, const double y[6], double dt, double eps, double yn[6]) {
  double f0[6], f1[6], yt[6];
  geodesic_rhs(a, M, y, eps, f0);
  for (int k = 0; k < 6; ++k) yt[k] = y[k] + f0[k] * dt;  // (14)
  for (int it = 0; it < K; ++it) {
    geodesic_rhs(a, M, yt, eps, f1);
    for (int k = 0; k < 6; ++k) yt[k] = y[k] + 0.5 * dt * (f1[k] + f0[k]);  // (15)
  }
  for (int k = 0; k < 6; ++k) yn[k] = yt[k];
}

// Particle shape function: first-order cloud-in-cell S^(x) = max(0, 1-|x|) "by
// default, but a third order spline is also available ... through a configuration option": the
// cubic B-spline  2/3 - x^2 + |x|^3/2 (|x| < 1),  (2-|x|)^3/6 (1 <= |x| < 2),  0 beyond.
// g_shape_order is that option (1 or 3), set by orc_set_shape_order; it selects the shape used
// by the gather, the current deposit and the charge density alike.
int shape_ext() { return g_shape_order == 3 ? 1 : 0; }   // extra nodes of support on each side
double shape(double x) {
  const double ax = std::fabs(x);
  if (g_shape_order == 3) {
    if (ax < 1.0) return 2.0 / 3.0 - ax * ax + 0.5 * ax * ax * ax;
    if (ax < 2.0) return (2.0 - ax) * (2.0 - ax) * (2.0 - ax) / 6.0;
    return 0.0;
  }
  return std::max(0.0, 1.0 - ax);
}

// ---------------------------------------------------------------------------
// Auxiliary fields (B9),(B11) and circulations (B8),(B10), PAPER.md:478-518,
// with the 1/2 restored in E_phi (reading G2) and Eq.(11) as the axis value of
// C_H^r (reading G4).  Every metric coefficient is evaluated at the location of
// the field it multiplies, then averaged.
// ---------------------------------------------------------------------------
struct Coef {
  double a_grr, a_gthth, a_gphph, a_grph, sg_beta;
};
Coef coef(const Grid& g, double i, double j) {
  Metric m = metric(g.a, g.M, g.r(i), g.th(j));
  return Coef{m.alpha * m.g_rr, m.alpha * m.g_thth, m.alpha * m.g_phph, m.alpha * m.g_rph,
              m.sqrtg * m.beta_r};
}

void circulation(const Grid& g, const double* ADr, const double* ADth, const double* ADph,
                 const double* ABr, const double* ABth, const double* ABph, const double* Dr,
                 const double* Dth, const double* Dph, const double* Br, const double* Bth,
                 const double* Bph, double* CHr, double* CHth, double* CHph, double* CEr,
                 double* CEth, double* CEph) {
  const size_t n = g.size();
  std::vector<double> Hr(n, 0.0), Hth(n, 0.0), Hph(n, 0.0), Er(n, 0.0), Eth(n, 0.0), Eph(n, 0.0);
  const int ilo = -g.G + 1, ihi = g.nr + g.G - 1;  // where both i-1 and i+1 are stored
#pragma omp parallel for schedule(static)          // row-parallel, no reduction: bit-identical to serial
  for (int j = 0; j <= g.nth; ++j)
    for (int i = ilo; i <= ihi; ++i) {
      const size_t k = g.idx(i, j);
      // node-in-theta components -------------------------------------------------
      // H_theta at (i+1/2, j)
      Hth[k] = coef(g, i + 0.5, j).a_gthth * Bth[k] +
               0.5 * (coef(g, i, j).sg_beta * Dph[g.idx(i, j)] +
                      coef(g, i + 1, j).sg_beta * Dph[g.idx(i + 1, j)]);
      // E_r at (i+1/2, j)
      Er[k] = coef(g, i + 0.5, j).a_grr * Dr[k] +
              0.5 * (coef(g, i, j).a_grph * Dph[g.idx(i, j)] +
                     coef(g, i + 1, j).a_grph * Dph[g.idx(i + 1, j)]);
      // E_phi at (i, j)   (1/2 restored on the last bracket)
      Eph[k] = coef(g, i, j).a_gphph * Dph[k] +
               0.5 * (coef(g, i + 0.5, j).a_grph * Dr[g.idx(i, j)] +
                      coef(g, i - 0.5, j).a_grph * Dr[g.idx(i - 1, j)]) +
               0.5 * (coef(g, i + 0.5, j).sg_beta * Bth[g.idx(i, j)] +
                      coef(g, i - 0.5, j).sg_beta * Bth[g.idx(i - 1, j)]);
      if (j == g.nth) continue;
      // half-in-theta components -------------------------------------------------
      // H_r at (i, j+1/2)
      Hr[k] = coef(g, i, j + 0.5).a_grr * Br[k] +
              0.5 * (coef(g, i + 0.5, j + 0.5).a_grph * Bph[g.idx(i, j)] +
                     coef(g, i - 0.5, j + 0.5).a_grph * Bph[g.idx(i - 1, j)]);
      // H_phi at (i+1/2, j+1/2)
      Hph[k] = coef(g, i + 0.5, j + 0.5).a_gphph * Bph[k] +
               0.5 * (coef(g, i, j + 0.5).a_grph * Br[g.idx(i, j)] +
                      coef(g, i + 1, j + 0.5).a_grph * Br[g.idx(i + 1, j)]) -
               0.5 * (coef(g, i, j + 0.5).sg_beta * Dth[g.idx(i, j)] +
                      coef(g, i + 1, j + 0.5).sg_beta * Dth[g.idx(i + 1, j)]);
      // E_theta at (i, j+1/2)
      Eth[k] = coef(g, i, j + 0.5).a_gthth * Dth[k] -
               0.5 * (coef(g, i + 0.5, j + 0.5).sg_beta * Bph[g.idx(i, j)] +
                      coef(g, i - 0.5, j + 0.5).sg_beta * Bph[g.idx(i - 1, j)]);
    }
  for (size_t k = 0; k < n; ++k) CHr[k] = CHth[k] = CHph[k] = CEr[k] = CEth[k] = CEph[k] = 0.0;
#pragma omp parallel for schedule(static)
  for (int j = 0; j <= g.nth; ++j)
    for (int i = 0; i <= g.nr; ++i) {
      const size_t k = g.idx(i, j);
      const double dr_node = g.r(i + 0.5) - g.r(i - 0.5);  // length of the r-edge centred on node i
      const double dr_half = g.r(i + 1) - g.r(i);          // length of the r-edge centred on i+1/2
      // (B8) D^r at (i+1/2, j), i < nr
      if (i < g.nr) {
        if (j == 0)  // Eq.(11): half face on the axis, only the theta=dth/2 side contributes
          CHr[k] = Hph[g.idx(i, 0)] * g.dphi / ADr[k];
        else if (j == g.nth)
          CHr[k] = -Hph[g.idx(i, g.nth - 1)] * g.dphi / ADr[k];
        else
          CHr[k] = (Hph[g.idx(i, j)] - Hph[g.idx(i, j - 1)]) * g.dphi / ADr[k];
      }
      // (B8) D^theta at (i, j+1/2)
      if (j < g.nth) CHth[k] = (Hph[g.idx(i - 1, j)] - Hph[g.idx(i, j)]) * g.dphi / ADth[k];
      // (B8) D^phi at (i, j); on the axes D^phi = 0 is imposed
      if (j > 0 && j < g.nth)
        CHph[k] = ((Hth[g.idx(i, j)] - Hth[g.idx(i - 1, j)]) * g.dth +
                   (Hr[g.idx(i, j - 1)] - Hr[g.idx(i, j)]) * dr_node) /
                  ADph[k];
      // (B10) B^r at (i, j+1/2)
      if (j < g.nth) CEr[k] = -(Eph[g.idx(i, j + 1)] - Eph[g.idx(i, j)]) * g.dphi / ABr[k];
      // (B10) B^theta at (i+1/2, j); B^theta = 0 on the axes
      if (i < g.nr && j > 0 && j < g.nth)
        CEth[k] = -(Eph[g.idx(i, j)] - Eph[g.idx(i + 1, j)]) * g.dphi / ABth[k];
      // (B10) B^phi at (i+1/2, j+1/2)
      if (i < g.nr && j < g.nth)
        CEph[k] = -((Eth[g.idx(i + 1, j)] - Eth[g.idx(i, j)]) * g.dth +
                    (Er[g.idx(i, j)] - Er[g.idx(i, j + 1)]) * dr_half) /
                  ABph[k];
    }
}

// Field boundary conditions (S8): axis values, radial guards =
// last physical value (the same closure is used at the outer edge
// underneath the damping layer), theta ghost rows by parity (for the gather).
void apply_bc(const Grid& g, double* Dr, double* Dth, double* Dph, double* Br, double* Bth,
              double* Bph) {
  struct C { double* F; const Stag* st; };
  C comps[6] = {{Dr, &ST_Dr}, {Dth, &ST_Dth}, {Dph, &ST_Dph}, {Br, &ST_Br}, {Bth, &ST_Bth}, {Bph, &ST_Bph}};
  for (int i = -g.G; i <= g.nr + g.G; ++i) {
    Dph[g.idx(i, 0)] = 0.0;
    Dph[g.idx(i, g.nth)] = 0.0;
    Bth[g.idx(i, 0)] = 0.0;
    Bth[g.idx(i, g.nth)] = 0.0;
  }
  for (auto& c : comps) {
    const int hi = (c.st->sr == 0.0) ? g.nr : g.nr - 1;
    const int jhi = (c.st->sth == 0.0) ? g.nth : g.nth - 1;
    for (int j = 0; j <= jhi; ++j) {
      for (int i = -g.G; i < 0; ++i) c.F[g.idx(i, j)] = c.F[g.idx(0, j)];
      for (int i = hi + 1; i <= g.nr + g.G; ++i) c.F[g.idx(i, j)] = c.F[g.idx(hi, j)];
    }
    for (int i = -g.G; i <= g.nr + g.G; ++i) {
      for (int j = -g.G; j < 0; ++j) c.F[g.idx(i, j)] = fetch(g, c.F, *c.st, i, j);
      for (int j = jhi + 1; j <= g.nth + g.G; ++j) c.F[g.idx(i, j)] = fetch(g, c.F, *c.st, i, j);
    }
  }
}

}  // namespace

// =============================================================================
// C entry points (ctypes)
// =============================================================================
extern "C" {

// out[23]: alpha, beta_r, g_rr, g_thth, g_phph, g_rph, gu_rr, gu_thth, gu_phph, gu_rph, sqrtg,
//          dr_alpha, dth_alpha, dr_beta, dth_beta, dr_gu_rr, dth_gu_rr, dr_gu_thth, dth_gu_thth,
//          dr_gu_phph, dth_gu_phph, dr_gu_rph, dth_gu_rph
void orc_metric(double a, double M, double r, double th, double* out) {
  Metric m = metric(a, M, r, th);
  const double v[23] = {m.alpha, m.beta_r, m.g_rr, m.g_thth, m.g_phph, m.g_rph, m.gu_rr,
                        m.gu_thth, m.gu_phph, m.gu_rph, m.sqrtg, m.dr_alpha, m.dth_alpha,
                        m.dr_beta, m.dth_beta, m.dr_gu_rr, m.dth_gu_rr, m.dr_gu_thth,
                        m.dth_gu_thth, m.dr_gu_phph, m.dth_gu_phph, m.dr_gu_rph, m.dth_gu_rph};
  std::memcpy(out, v, sizeof v);
}

void orc_gauss_legendre(int n, double* x, double* w) { gauss_legendre(n, x, w); }

void orc_grid_shape(const orc_params* p, int32_t* nrp, int32_t* nthp) {
  Grid g(*p);
  *nrp = g.NRP;
  *nthp = g.NTHP;
}

void orc_areas(const orc_params* p, double* ADr, double* ADth, double* ADph, double* ABr,
               double* ABth, double* ABph) {
  compute_areas(Grid(*p), ADr, ADth, ADph, ABr, ABth, ABph);
}

// Gather D^i, B^i at (x1 = ln r, x2 = theta); out[6] = Dr,Dth,Dph,Br,Bth,Bph.
void orc_gather(const orc_params* p, const double* Dr, const double* Dth, const double* Dph,
                const double* Br, const double* Bth, const double* Bph, double x1, double x2,
                double* out) {
  Grid g(*p);
  const double fx = (x1 - g.xi_in) / g.dxi, fy = x2 / g.dth;
  out[0] = gather1(g, Dr, ST_Dr, fx, fy);
  out[1] = gather1(g, Dth, ST_Dth, fx, fy);
  out[2] = gather1(g, Dph, ST_Dph, fx, fy);
  out[3] = gather1(g, Br, ST_Br, fx, fy);
  out[4] = gather1(g, Bth, ST_Bth, fx, fy);
  out[5] = gather1(g, Bph, ST_Bph, fx, fy);
}

void orc_boris(double a, double M, double r, double th, const double* u, const double* D,
               const double* B, double sgn, double dt, double* uout) {
  boris(metric(a, M, r, th), u, D, B, sgn, dt, uout);
}
void orc_vay(double a, double M, double r, double th, const double* u, const double* D,
             const double* B, double sgn, double dt, double* uout) {
  vay(metric(a, M, r, th), u, D, B, sgn, dt, uout);
}
// momentum update used by orc_push (0 = Boris, 1 = Vay); returns the previous value
int orc_set_pusher(int which) {
  const int old = g_pusher;
  if (which == 0 || which == 1) g_pusher = which;
  return old;
}

void orc_geodesic_rhs(double a, double M, const double* y, double eps, double* f) {
  geodesic_rhs(a, M, y, eps, f);
}
void orc_geodesic(double a, double M, int K, const double* y, double dt, double eps, double* yn) {
  geodesic(a, M, K, y, dt, eps, yn);
}
// nsteps geodesic steps of one particle, state recorded every `every` steps into traj[.][6]
void orc_geodesic_traj(double a, double M, int K, const double* y0, double dt, double eps,
                       int64_t nsteps, int64_t every, double* traj) {
  double y[6], yn[6];
  std::memcpy(y, y0, sizeof y);
  int64_t rec = 0;
  for (int64_t n = 0; n < nsteps; ++n) {
    if (n % every == 0) std::memcpy(traj + 6 * (rec++), y, sizeof y);
    geodesic(a, M, K, y, dt, eps, yn);
    std::memcpy(y, yn, sizeof y);
  }
}

// One particle step S4: gather D^n,B^n at x^n -> full-dt
// Boris (PAPER.md:204 bundled half steps) -> geodesic -> x1 = ln r -> axis
// reflection -> removal flag and new cell.
// flag bit0: 1 = positron (q/m=+1), 0 = electron (q/m=-1); bit1: removed;
// bit2: photon species (PAPER.md:153 "eps = 0 in u^0", :155 "photons ... only the geodesic
// part"): no gather, no Boris, geodesic with eps = 0; carries no charge (no current, no rho).
// x2dep = un-reflected new theta, used by the deposit (reading G13).
// Particles whose removed bit is already set are copied through unchanged.
void orc_push(const orc_params* p, const double* Dr, const double* Dth, const double* Dph,
              const double* Br, const double* Bth, const double* Bph, int64_t n, const double* x1,
              const double* x2, const double* x3, const double* u1, const double* u2,
              const double* u3, const uint32_t* flag, double dt, double* x1n, double* x2n,
              double* x3n, double* u1n, double* u2n, double* u3n, double* x2dep, uint32_t* celln,
              uint32_t* flagn) {
  const Grid g(*p);
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < n; ++k) {
    if (flag[k] & 2u) {
      x1n[k] = x1[k]; x2n[k] = x2[k]; x3n[k] = x3[k];
      u1n[k] = u1[k]; u2n[k] = u2[k]; u3n[k] = u3[k];
      x2dep[k] = x2[k]; celln[k] = 0xFFFFFFFFu; flagn[k] = flag[k];
      continue;
    }
    const bool photon = (flag[k] & 4u) != 0;
    const double sgn = (flag[k] & 1u) ? 1.0 : -1.0;
    const double r = std::exp(x1[k]), th = x2[k];
    const double u[3] = {u1[k], u2[k], u3[k]};
    double ub[3] = {u[0], u[1], u[2]};
    if (!photon) {
      const double fx = (x1[k] - g.xi_in) / g.dxi, fy = th / g.dth;
      double D[3], B[3];
      D[0] = gather1(g, Dr, ST_Dr, fx, fy);
      D[1] = gather1(g, Dth, ST_Dth, fx, fy);
      D[2] = gather1(g, Dph, ST_Dph, fx, fy);
      B[0] = gather1(g, Br, ST_Br, fx, fy);
      B[1] = gather1(g, Bth, ST_Bth, fx, fy);
      B[2] = gather1(g, Bph, ST_Bph, fx, fy);
      if (g_pusher == 1) vay(metric(g.a, g.M, r, th), u, D, B, sgn, dt, ub);
      else boris(metric(g.a, g.M, r, th), u, D, B, sgn, dt, ub);
    }
    const double y[6] = {r, th, x3[k], ub[0], ub[1], ub[2]};
    double yn[6];
    geodesic(g.a, g.M, p->geo_iters, y, dt, photon ? 0.0 : 1.0, yn);
    const double xi_new = std::log(yn[0]);
    double thn = yn[1], uth = yn[4];
    x2dep[k] = thn;
    if (thn < 0.0) { thn = -thn; uth = -uth; }
    if (thn > M_PI) { thn = 2.0 * M_PI - thn; uth = -uth; }
    x1n[k] = xi_new; x2n[k] = thn; x3n[k] = yn[2];
    u1n[k] = yn[3]; u2n[k] = uth; u3n[k] = yn[5];
    const bool out = (xi_new < g.xi_in) || (xi_new >= p->xi_out);
    if (out) {
      flagn[k] = flag[k] | 2u;
      celln[k] = 0xFFFFFFFFu;
    } else {
      flagn[k] = flag[k];
      int ic = (int)std::floor((xi_new - g.xi_in) / g.dxi);
      int jc = (int)std::floor(thn / g.dth);
      ic = std::min(std::max(ic, 0), g.nr - 1);
      jc = std::min(std::max(jc, 0), g.nth - 1);
      celln[k] = (uint32_t)(jc * g.nr + ic);
    }
  }
}

// Charge-conserving deposit, Eq.(21)-(23) PAPER.md:208-233 with CIC shape.
// Accumulates the FLUXES F_r = J^r A^D_r at (i+1/2,j), F_th = J^th A^D_th at (i,j+1/2),
// F_ph = J^ph dV at (i,j) (+=).  Positions: old (x1o,x2o,x3o), new (x1n, x2dep
// un-reflected, x3n).  flag = flags BEFORE the step (particles already removed are
// skipped).  The per-particle prefix sum runs over exactly the nodes its two shape
// functions touch.
void orc_deposit(const orc_params* p, int64_t n, const double* x1o, const double* x2o,
                 const double* x3o, const double* x1n, const double* x2dep, const double* x3n,
                 const double* w, const uint32_t* flag, double dt, double* Fr, double* Fth,
                 double* Fph) {
  const Grid g(*p);
  for (int64_t k = 0; k < n; ++k) {
    if (flag[k] & (2u | 4u)) continue;                 // removed, or photon (no charge)
    const double Q = ((flag[k] & 1u) ? 1.0 : -1.0) * w[k];
    const double xa = (x1o[k] - g.xi_in) / g.dxi, xb = (x1n[k] - g.xi_in) / g.dxi;
    const double ya = x2o[k] / g.dth, yb = x2dep[k] / g.dth;
    const int ext = shape_ext();
    const int ilo = (int)std::floor(std::min(xa, xb)) - ext, ihi = (int)std::floor(std::max(xa, xb)) + 1 + ext;
    const int jlo = (int)std::floor(std::min(ya, yb)) - ext, jhi = (int)std::floor(std::max(ya, yb)) + 1 + ext;
    // (22) without /dV:  W_r,ij and W_th,ij
    for (int j = jlo; j <= jhi; ++j) {
      double acc = 0.0;  // F_r(ilo-1/2, j) = 0
      for (int i = ilo; i < ihi; ++i) {
        const double Wr = 0.5 * Q *
                          (shape(xb - i) * shape(yb - j) - shape(xa - i) * shape(yb - j) +
                           shape(xb - i) * shape(ya - j) - shape(xa - i) * shape(ya - j));
        acc -= Wr / dt;  // (21): F_r(i+1/2) = F_r(i-1/2) - W_r,i/dt
        Fr[g.idx(i, j)] += acc;
      }
    }
    for (int i = ilo; i <= ihi; ++i) {
      double acc = 0.0;
      for (int j = jlo; j < jhi; ++j) {
        const double Wth = 0.5 * Q *
                           (shape(xb - i) * shape(yb - j) - shape(xb - i) * shape(ya - j) +
                            shape(xa - i) * shape(yb - j) - shape(xa - i) * shape(ya - j));
        acc -= Wth / dt;
        Fth[g.idx(i, j)] += acc;
      }
    }
    // (23), sign/normalisation reading G5
    const double vphi = Q * (x3n[k] - x3o[k]) / dt;
    for (int j = jlo; j <= jhi; ++j)
      for (int i = ilo; i <= ihi; ++i) {
        const double S = (1.0 / 3.0) * shape(xb - i) * shape(yb - j) +
                         (1.0 / 6.0) * shape(xb - i) * shape(ya - j) +
                         (1.0 / 6.0) * shape(xa - i) * shape(yb - j) +
                         (1.0 / 3.0) * shape(xa - i) * shape(ya - j);
        Fph[g.idx(i, j)] += vphi * S;
      }
  }
}

// Fold the theta-ghost rows onto their mirror rows (reading G13): even parity for
// node-located scalars/fluxes F_r, F_ph, rho*dV; odd for F_th.  Ghost rows are zeroed.
static void fold_rows(const Grid& g, double* F, bool half_in_theta, double parity) {
  for (int gh = 1; gh <= g.G; ++gh)
    for (int i = -g.G; i <= g.nr + g.G; ++i) {
      if (!half_in_theta) {
        F[g.idx(i, gh)] += parity * F[g.idx(i, -gh)];
        F[g.idx(i, g.nth - gh)] += parity * F[g.idx(i, g.nth + gh)];
        F[g.idx(i, -gh)] = 0.0;
        F[g.idx(i, g.nth + gh)] = 0.0;
      } else {
        F[g.idx(i, gh - 1)] += parity * F[g.idx(i, -gh)];
        F[g.idx(i, g.nth - gh)] += parity * F[g.idx(i, g.nth - 1 + gh)];
        F[g.idx(i, -gh)] = 0.0;
        F[g.idx(i, g.nth - 1 + gh)] = 0.0;
      }
    }
  if (half_in_theta)  // row nth+G is outside the half-staggered range: clear it
    for (int i = -g.G; i <= g.nr + g.G; ++i) F[g.idx(i, g.nth + g.G)] = 0.0;
}

// One (1,2,1)x(1,2,1)/16 pass in index space (S10; BASELINE.json config 5; not in
// the paper).  theta neighbours across the axis by parity, radial neighbours beyond
// the stored range clamped.
static void filter_pass(const Grid& g, double* F, bool half_in_theta, double parity) {
  const int jhi = half_in_theta ? g.nth - 1 : g.nth;
  std::vector<double> tmp(g.size(), 0.0);
  auto at = [&](int i, int j) -> double {
    i = std::min(std::max(i, -g.G), g.nr + g.G);
    double sign = 1.0;
    if (!half_in_theta) {
      if (j < 0) { j = -j; sign = parity; }
      if (j > jhi) { j = 2 * g.nth - j; sign = parity; }
    } else {
      if (j < 0) { j = -1 - j; sign = parity; }
      if (j > jhi) { j = 2 * g.nth - 1 - j; sign = parity; }
    }
    return sign * F[g.idx(i, j)];
  };
  for (int j = 0; j <= jhi; ++j)
    for (int i = -g.G; i <= g.nr + g.G; ++i) {
      double s = 0.0;
      const double wgt[3] = {1.0, 2.0, 1.0};
      for (int dj = -1; dj <= 1; ++dj)
        for (int di = -1; di <= 1; ++di) s += wgt[dj + 1] * wgt[di + 1] * at(i + di, j + dj);
      tmp[g.idx(i, j)] = s / 16.0;
    }
  for (int j = 0; j <= jhi; ++j)
    for (int i = -g.G; i <= g.nr + g.G; ++i) F[g.idx(i, j)] = tmp[g.idx(i, j)];
}

// Fold ghosts, optional filter passes on the fluxes, then J^r = F_r/A^D_r,
// J^th = F_th/A^D_th, J^ph = F_ph/dV with dV = dphi*A^D_ph (S5/S10).
void orc_finalize_current(const orc_params* p, double* Fr, double* Fth, double* Fph,
                          int filter_passes) {
  const Grid g(*p);
  std::vector<double> ADr(g.size()), ADth(g.size()), ADph(g.size()), ABr(g.size()), ABth(g.size()),
      ABph(g.size());
  compute_areas(g, ADr.data(), ADth.data(), ADph.data(), ABr.data(), ABth.data(), ABph.data());
  fold_rows(g, Fr, false, +1.0);
  fold_rows(g, Fph, false, +1.0);
  fold_rows(g, Fth, true, -1.0);
  for (int pass = 0; pass < filter_passes; ++pass) {
    filter_pass(g, Fr, false, +1.0);
    filter_pass(g, Fph, false, +1.0);
    filter_pass(g, Fth, true, -1.0);
  }
  for (size_t k = 0; k < g.size(); ++k) {
    Fr[k] = (ADr[k] > 0.0) ? Fr[k] / ADr[k] : 0.0;
    Fth[k] = (ADth[k] > 0.0) ? Fth[k] / ADth[k] : 0.0;
    Fph[k] = (ADph[k] > 0.0) ? Fph[k] / (g.dphi * ADph[k]) : 0.0;
  }
}

// Only the fold (for the continuity test, which works on fluxes and rho*dV).
void orc_fold_current(const orc_params* p, double* Fr, double* Fth, double* Fph) {
  const Grid g(*p);
  fold_rows(g, Fr, false, +1.0);
  fold_rows(g, Fph, false, +1.0);
  fold_rows(g, Fth, true, -1.0);
}

// rho*dV on vertices: rhoV_ij = sum Q S_ij(x), folded (S6).  If divide != 0 the
// result is divided by dV_ij = dphi*A^D_ph,ij to give rho.
void orc_rho(const orc_params* p, int64_t n, const double* x1, const double* x2, const double* w,
             const uint32_t* flag, int divide, double* rho) {
  const Grid g(*p);
  for (size_t k = 0; k < g.size(); ++k) rho[k] = 0.0;
  for (int64_t k = 0; k < n; ++k) {
    if (flag[k] & (2u | 4u)) continue;                 // removed, or photon (no charge)
    const double Q = ((flag[k] & 1u) ? 1.0 : -1.0) * w[k];
    const double x = (x1[k] - g.xi_in) / g.dxi, y = x2[k] / g.dth;
    const int i0 = (int)std::floor(x), j0 = (int)std::floor(y);
    const int ext = shape_ext();
    for (int j = j0 - ext; j <= j0 + 1 + ext; ++j)
      for (int i = i0 - ext; i <= i0 + 1 + ext; ++i) rho[g.idx(i, j)] += Q * shape(x - i) * shape(y - j);
  }
  fold_rows(g, rho, false, +1.0);
  if (divide) {
    std::vector<double> ADr(g.size()), ADth(g.size()), ADph(g.size()), ABr(g.size()),
        ABth(g.size()), ABph(g.size());
    compute_areas(g, ADr.data(), ADth.data(), ADph.data(), ABr.data(), ABth.data(), ABph.data());
    for (size_t k = 0; k < g.size(); ++k)
      rho[k] = (ADph[k] > 0.0) ? rho[k] / (g.dphi * ADph[k]) : 0.0;
  }
}

void orc_apply_bc(const orc_params* p, double* Dr, double* Dth, double* Dph, double* Br,
                  double* Bth, double* Bph) {
  apply_bc(Grid(*p), Dr, Dth, Dph, Br, Bth, Bph);
}

void orc_circulation(const orc_params* p, const double* Dr, const double* Dth, const double* Dph,
                     const double* Br, const double* Bth, const double* Bph, double* CHr,
                     double* CHth, double* CHph, double* CEr, double* CEth, double* CEph) {
  const Grid g(*p);
  std::vector<double> ADr(g.size()), ADth(g.size()), ADph(g.size()), ABr(g.size()), ABth(g.size()),
      ABph(g.size());
  compute_areas(g, ADr.data(), ADth.data(), ADph.data(), ABr.data(), ABth.data(), ABph.data());
  circulation(g, ADr.data(), ADth.data(), ADph.data(), ABr.data(), ABth.data(), ABph.data(), Dr,
              Dth, Dph, Br, Bth, Bph, CHr, CHth, CHph, CEr, CEth, CEph);
}

// Semi-implicit predictor-corrector field update, Eq.(9),(10) PAPER.md:113-128 with
// the factor reading G3 (dt*(alpha_i C^n + beta_i C~), alpha_i = 1 - beta_i), N =
// field_iters correctors, BCs (S8) on every iterate, damping (S9) after the step.
// D,B in-out (6 arrays); J = current densities (3 arrays, may be null = vacuum);
// bg = background fields for the damping layer (6 arrays, null = damp to zero).
void orc_field_step(const orc_params* p, double* Dr, double* Dth, double* Dph, double* Br,
                    double* Bth, double* Bph, const double* Jr, const double* Jth,
                    const double* Jph, const double* const* bg, double dt) {
  const Grid g(*p);
  const size_t n = g.size();
  std::vector<double> ADr(n), ADth(n), ADph(n), ABr(n), ABth(n), ABph(n);
  compute_areas(g, ADr.data(), ADth.data(), ADph.data(), ABr.data(), ABth.data(), ABph.data());
  double* F[6] = {Dr, Dth, Dph, Br, Bth, Bph};
  const double* J[3] = {Jr, Jth, Jph};
  apply_bc(g, F[0], F[1], F[2], F[3], F[4], F[5]);
  std::vector<std::vector<double>> Cn(6, std::vector<double>(n)), Ct(6, std::vector<double>(n)),
      It(6, std::vector<double>(n));
  auto circ = [&](double* const* X, std::vector<std::vector<double>>& C) {
    circulation(g, ADr.data(), ADth.data(), ADph.data(), ABr.data(), ABth.data(), ABph.data(),
                X[0], X[1], X[2], X[3], X[4], X[5], C[0].data(), C[1].data(), C[2].data(),
                C[3].data(), C[4].data(), C[5].data());
  };
  auto physical = [&](int c, int i, int j) -> bool {
    static const Stag* st[6] = {&ST_Dr, &ST_Dth, &ST_Dph, &ST_Br, &ST_Bth, &ST_Bph};
    const int ihi = (st[c]->sr == 0.0) ? g.nr : g.nr - 1;
    const int jhi = (st[c]->sth == 0.0) ? g.nth : g.nth - 1;
    return i >= 0 && i <= ihi && j >= 0 && j <= jhi;
  };
  double* itp[6];
  for (int c = 0; c < 6; ++c) {
    It[c].assign(F[c], F[c] + n);
    itp[c] = It[c].data();
  }
  circ(F, Cn);
  // predictor (9)
  for (int c = 0; c < 6; ++c)
    for (int j = 0; j <= g.nth; ++j)
      for (int i = 0; i <= g.nr; ++i) {
        if (!physical(c, i, j)) continue;
        const size_t k = g.idx(i, j);
        const double Jk = (c < 3 && J[c]) ? J[c][k] : 0.0;
        It[c][k] = F[c][k] + (Cn[c][k] - Jk) * dt;
      }
  apply_bc(g, itp[0], itp[1], itp[2], itp[3], itp[4], itp[5]);
  // correctors (10)
  const double bi = p->beta_impl, ai = 1.0 - p->beta_impl;
  for (int it = 0; it < p->field_iters; ++it) {
    circ(itp, Ct);
    for (int c = 0; c < 6; ++c)
      for (int j = 0; j <= g.nth; ++j)
        for (int i = 0; i <= g.nr; ++i) {
          if (!physical(c, i, j)) continue;
          const size_t k = g.idx(i, j);
          const double Jk = (c < 3 && J[c]) ? J[c][k] : 0.0;
          It[c][k] = F[c][k] + dt * (ai * Cn[c][k] + bi * Ct[c][k]) - Jk * dt;
        }
    apply_bc(g, itp[0], itp[1], itp[2], itp[3], itp[4], itp[5]);
  }
  // damping layer (S9, reading G14): outer damp_cells radial indices
  if (p->damp_cells > 0) {
    const int i0 = g.nr - p->damp_cells;
    for (int c = 0; c < 6; ++c)
      for (int j = 0; j <= g.nth; ++j)
        for (int i = i0 + 1; i <= g.nr; ++i) {
          if (!physical(c, i, j)) continue;
          const size_t k = g.idx(i, j);
          const double s = (double)(i - i0) / (double)(g.nr - i0);
          const double lam = 1.0 - p->damp_coef * s * s * s;
          const double b = bg ? bg[c][k] : 0.0;
          It[c][k] = b + (It[c][k] - b) * lam;
        }
    apply_bc(g, itp[0], itp[1], itp[2], itp[3], itp[4], itp[5]);
  }
  for (int c = 0; c < 6; ++c) std::memcpy(F[c], It[c].data(), n * sizeof(double));
}

// S11: stable sort by key = removed ? 0xFFFFFFFF : cell.  perm[k] = source index.
void orc_sort(int64_t n, const uint32_t* cell, const uint32_t* flag, uint32_t* perm) {
  std::vector<uint32_t> key(n);
  for (int64_t k = 0; k < n; ++k) key[k] = (flag[k] & 2u) ? 0xFFFFFFFFu : cell[k];
  std::iota(perm, perm + n, 0u);
  std::stable_sort(perm, perm + n, [&](uint32_t x, uint32_t y) { return key[x] < key[y]; });
}

// S11b (not in the paper; BASELINE.json north_star "deposition ... keyed by sorted cell", DESIGN.md
// reading S11b): the contention-free cell order.  With rank = position of a particle among the
// particles of its cell in the stable order of S11, live particles are ordered by the tuple
// (cell / B, rank, cell % B); removed particles follow in their input order.  All tuples differ,
// so the order is unique.  Written out as the definition: S11, ranks, then a sort by the tuple.
void orc_sort_interleaved(int64_t n, const uint32_t* cell, const uint32_t* flag, uint32_t ncells,
                          uint32_t B, uint32_t* perm) {
  std::vector<uint32_t> key(n), stable(n), rank(n);
  for (int64_t k = 0; k < n; ++k) key[k] = (flag[k] & 2u) ? ncells : std::min(cell[k], ncells);
  std::iota(stable.begin(), stable.end(), 0u);
  std::stable_sort(stable.begin(), stable.end(), [&](uint32_t x, uint32_t y) { return key[x] < key[y]; });
  for (int64_t k = 0, r = 0; k < n; ++k) {          // rank of the particle at sorted position k
    r = (k > 0 && key[stable[k]] == key[stable[k - 1]]) ? r + 1 : 0;
    rank[stable[k]] = (uint32_t)r;
  }
  std::copy(stable.begin(), stable.end(), perm);
  auto before = [&](uint32_t x, uint32_t y) {
    const bool rx = key[x] >= ncells, ry = key[y] >= ncells;
    if (rx || ry) return !rx && ry;                  // live before removed; removed keep their order
    if (key[x] / B != key[y] / B) return key[x] / B < key[y] / B;
    if (rank[x] != rank[y]) return rank[x] < rank[y];
    return key[x] % B < key[y] % B;
  };
  std::stable_sort(perm, perm + n, before);
}

// S12: order-preserving removal of flagged particles; idx[0..count) = surviving
// source indices in order; returns count.
int64_t orc_compact(int64_t n, const uint32_t* flag, uint32_t* idx) {
  int64_t c = 0;
  for (int64_t k = 0; k < n; ++k)
    if (!(flag[k] & 2u)) idx[c++] = (uint32_t)k;
  return c;
}

// ---------------------------------------------------------------------------
// Simplified pair production of Section 4 (Eq.26).  Counter-based random
// numbers: Philox4x32-10 (Salmon et al. 2011), written out from the published round function;
// pinned by the known-answer vectors in tests/golden/philox4x32_10.txt.
// ---------------------------------------------------------------------------
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
// uniform in [0,1) with 53 bits from the first two words; counter = (index lo, index hi, step, 0)
double orc_uniform(uint64_t seed, uint32_t step, uint64_t index) {
  const uint32_t ctr[4] = {(uint32_t)index, (uint32_t)(index >> 32), step, 0u};
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t o[4];
  orc_philox4x32_10(ctr, key, o);
  const uint64_t bits = (((uint64_t)o[0] << 32) | o[1]) >> 11;
  return (double)bits * (1.0 / 9007199254740992.0);
}

// One pair-production pass over particles [0, n) (arrays have room for `capacity`), in the
// paper's words plus the readings P1-P4 of DESIGN.md:
//  * a lepton whose FIDO Lorentz factor Gamma = alpha u^0 = sqrt(1 + gamma^ij u_i u_j) reaches
//    gamma_thr emits ONE photon of FIDO energy eps_ph "in the same direction": photon
//    u_i = u_i eps_ph/|u| with |u| = sqrt(gamma^ij u_i u_j); the lepton keeps the rest of its
//    momentum, u_i <- u_i (1 - eps_ph/|u|) (P1; only if |u| > eps_ph);
//  * a photon converts with probability p_convert = 1 - exp(-tau dt) (Eq.26; the caller passes
//    the number), decided by U(seed, step, index) < p_convert (P2); "each particle gets exactly
//    half of the photon energy": E = |u| is the photon's FIDO energy now, each lepton gets
//    Gamma = E/2 along the photon's direction, |u_l| = sqrt(Gamma^2 - 1) (P3; only if E/2 > 1).
//    The photon's slot becomes the electron, the positron is a new particle;
//  * new particles (photons, positrons) inherit position, cell and weight and are appended at
//    n, n+1, ... in the order of their parents (P4).  Returns the new count (<= capacity;
//    events whose child would not fit do not happen (P5) and *overflow is set).
int64_t orc_pair_production(const orc_params* p, int64_t n, int64_t capacity, double* x1, double* x2,
                            double* x3, double* u1, double* u2, double* u3, double* w, uint32_t* cell,
                            uint32_t* flag, double gamma_thr, double eps_ph, double p_convert,
                            uint64_t seed, uint32_t step, int32_t* overflow) {
  int64_t m = n;
  *overflow = 0;
  for (int64_t k = 0; k < n; ++k) {
    if (flag[k] & 2u) continue;
    const Metric g = metric(p->a, p->M, std::exp(x1[k]), x2[k]);
    const double u[3] = {u1[k], u2[k], u3[k]};
    const double N = norm_up(g, u);
    double child_scale = 0.0, parent_scale = 1.0;
    uint32_t child_flag = 0, parent_flag = flag[k];
    if (!(flag[k] & 4u)) {                             // lepton: emission
      const double Gamma = std::sqrt(1.0 + N), umag = std::sqrt(N);
      if (Gamma >= gamma_thr && umag > eps_ph) {
        child_scale = eps_ph / umag;
        parent_scale = 1.0 - eps_ph / umag;
        child_flag = 4u;
      }
    } else {                                           // photon: conversion
      const double E = std::sqrt(N), Gl = 0.5 * E;
      if (orc_uniform(seed, step, (uint64_t)k) < p_convert && Gl > 1.0) {
        child_scale = parent_scale = std::sqrt(Gl * Gl - 1.0) / E;
        parent_flag = 0u;                              // electron
        child_flag = 1u;                               // positron
      }
    }
    if (child_scale == 0.0) continue;
    if (m >= capacity) {                               // P5: an event whose child has no room does not
      *overflow = 1;                                   // happen (the parent keeps momentum and species:
      continue;                                        // no charge or momentum is lost silently)
    }
    x1[m] = x1[k]; x2[m] = x2[k]; x3[m] = x3[k];
    u1[m] = u[0] * child_scale; u2[m] = u[1] * child_scale; u3[m] = u[2] * child_scale;
    w[m] = w[k]; cell[m] = cell[k]; flag[m] = child_flag;
    ++m;
    u1[k] = u[0] * parent_scale; u2[k] = u[1] * parent_scale; u3[k] = u[2] * parent_scale;
    flag[k] = parent_flag;
  }
  return m;
}

// Boyer-Lindquist / FIDO diagnostics of a Kerr-Schild particle state ((A6), (A7)).
// out[4] = { E_inf = -u_t, Gamma_FIDO = alpha u^0, u_r^BL, phi_BL }.
//   -u_t = alpha^2 u^0 - beta^r u_r                      (u_t = g_{t mu} u^mu in the 3+1 split)
//   (A6) dt_KS = dt_BL + 2Mr/Delta dr, dphi_KS = dphi_BL + a/Delta dr  =>  covariant components transform
//   with the transposed Jacobian: u_r^BL = u_r^KS + (2Mr/Delta) u_t + (a/Delta) u_phi, others unchanged.
//   (A7) phi_KS = phi_BL + a/(2 sqrt(M^2-a^2)) ln|(r - r_+)/(r - r_-)|.
void orc_ks_to_bl(double a, double M, double x1, double th, double ph, const double u[3], double eps,
                  double* out) {
  const double r = std::exp(x1);
  const Metric m = metric(a, M, r, th);
  const double u0 = std::sqrt(eps + norm_up(m, u)) / m.alpha;
  const double E = m.alpha * m.alpha * u0 - m.beta_r * u[0];
  const double Delta = r * r - 2.0 * M * r + a * a;
  const double root = std::sqrt(M * M - a * a);
  out[0] = E;
  out[1] = m.alpha * u0;
  out[2] = u[0] + (2.0 * M * r / Delta) * (-E) + (a / Delta) * u[2];
  out[3] = ph - (root > 0.0 ? a / (2.0 * root) * std::log(std::fabs((r - (M + root)) / (r - (M - root)))) : 0.0);
}

double orc_shape(double x) { return shape(x); }
// shape order option (1 = cloud-in-cell, 3 = cubic B-spline); returns the previous value
int orc_set_shape_order(int order) {
  const int old = g_shape_order;
  if (order == 1 || order == 3) g_shape_order = order;
  return old;
}

// number of OpenMP threads of the parallel loops (particles in orc_push; grid rows in the areas
// and circulations); returns the previous value.  Used by the bit-identity test and the baseline.
int orc_set_num_threads(int n) {
#ifdef _OPENMP
  const int old = omp_get_max_threads();
  if (n > 0) omp_set_num_threads(n);
  return old;
#else
  (void)n;
  return 1;
#endif
}

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
