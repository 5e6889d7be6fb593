// Device arithmetic shared by the particle kernels of libgrpic.so (push_deposit.cu: first-order
// shape, tuned; push_spline3.cu: third-order shape): Kerr-Schild position terms with one
// reciprocal per point, right-hand sides of Eq.(12), generalised Boris (Eq.16-19), small-angle
// sin/cos update, and the exact general-window first-order deposit.  Closed forms: Appendix A
// with M restored.
#pragma once
#include <math.h>

#include "grpic_internal.cuh"
#include "poly_tables.cuh"

namespace {

// ---- the kernel's own exp / sincos: the algorithms of any libm (Cody-Waite reduction with a
// round-to-nearest magic constant, Horner polynomials), coefficients from the PolyTab kernel
// parameter (one LDCU each; a literal costs two UMOV on sm_100a), no special-case branches: arguments
// are ln r in [xi_in, xi_out] and theta near [0, pi]; anything else (NaN, huge) yields a
// non-finite or meaningless value that the caller's removal test catches.  Errors < 1 ulp.
constexpr double kMagic = 6755399441055744.0;        // 1.5 * 2^52: x + kMagic rounds x to an integer
__device__ __forceinline__ double exp_pt(const PolyTab& pt, double x) {
  const double t = fma(x, pt.v[kL2E], kMagic);
  const int n = __double2loint(t);
  const double fn = t - kMagic;
  double r = fma(fn, -pt.v[kLN2_HI], x);
  r = fma(fn, -pt.v[kLN2_LO], r);
  double p = pt.v[kEXP0];
  p = fma(p, r, pt.v[kEXP1]);
  p = fma(p, r, pt.v[kEXP2]);
  p = fma(p, r, pt.v[kEXP3]);
  p = fma(p, r, pt.v[kEXP4]);
  p = fma(p, r, pt.v[kEXP5]);
  p = fma(p, r, pt.v[kEXP6]);
  p = fma(p, r, pt.v[kEXP7]);
  p = fma(p, r, pt.v[kEXP8]);
  p = fma(p, r, pt.v[kEXP9]);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);                                 // exp(r), |r| <= ln2/2
  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));   // * 2^n
}
__device__ __forceinline__ void sincos_pt(const PolyTab& pt, double x, double& s, double& c) {
  const double t = fma(x, pt.v[kTWO_OVER_PI], kMagic);
  const int q = __double2loint(t);
  const double fk = t - kMagic;
  double r = fma(fk, -pt.v[kPIO2_1], x);
  r = fma(fk, -pt.v[kPIO2_2], r);
  r = fma(fk, -pt.v[kPIO2_3], r);                      // |r| <= pi/4
  const double z = r * r;
  double ps = fma(pt.v[kSIN0], z, pt.v[kSIN1]);
  double pc = fma(pt.v[kCOS0], z, pt.v[kCOS1]);
  ps = fma(ps, z, pt.v[kSIN2]);
  pc = fma(pc, z, pt.v[kCOS2]);
  ps = fma(ps, z, pt.v[kSIN3]);
  pc = fma(pc, z, pt.v[kCOS3]);
  ps = fma(ps, z, pt.v[kSIN4]);
  pc = fma(pc, z, pt.v[kCOS4]);
  ps = fma(ps, z, pt.v[kSIN5]);
  pc = fma(pc, z, pt.v[kCOS5]);
  const double sr = fma(ps * z, r, r);                // sin r
  const double cr = fma(pc * z, z, fma(z, -0.5, 1.0));   // cos r
  // quadrant q mod 4: (sin, cos) = (sr, cr), (cr, -sr), (-sr, -cr), (-cr, sr)
  const bool odd = (q & 1) != 0;
  const double sa = odd ? cr : sr, ca = odd ? sr : cr;
  s = __hiloint2double(__double2hiint(sa) ^ ((q << 30) & 0x80000000), __double2loint(sa));
  c = __hiloint2double(__double2hiint(ca) ^ (((q + 1) << 30) & 0x80000000), __double2loint(ca));
}

// 1/x: MUFU.RCP64H seed (relative error <= 2^-23, PTX rcp.approx.ftz.f64) + ONE third-order step
// y (1 + e + e^2), e = 1 - x y: error ~ e^3 = 2^-69, three FMAs instead of the four of two Newton
// steps; no special-case slow path.
__device__ __forceinline__ double rcp_nr(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);
  return fma(y, fma(e, e, e), y);
}
// 1/sqrt(x): MUFU.RSQ64H seed + one third-order step y (1 + e + 3/2 e^2), e = (1 - x y^2)/2.
__device__ __forceinline__ double rsqrt_nr(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double h = 0.5 * x;
  const double e = fma(-(h * y), y, 0.5);
  return fma(y, fma(e * 1.5, e, e), y);               // immediates only: no constant register pair
}

struct Pos {          // position-only terms at (r, theta)
  double r, s, c;     // r, sin, cos
  double rho2;
  double R;           // 1/rho^2
  double is2;         // 1/sin^2
  double beta;        // beta^r = 2Mr/(rho^2+2Mr)
  double zp1;         // 1+z
  double h;           // 1/(1+z) = alpha^2
  double r2a2;        // r^2 + a^2
  double r2;          // r^2
  double sc2;         // 2 sin cos
};

__device__ __forceinline__ Pos make_pos(const GridDev& g, double r, double s, double c) {
  Pos p;
  p.r = r; p.s = s; p.c = c;
  const double r2 = r * r;
  p.rho2 = fma(g.a2 * c, c, r2);
  const double twoMr = g.twoM * r;
  const double B = p.rho2 + twoMr;          // rho^2 (1+z)
  const double s2 = s * s;
  const double rb = p.rho2 * B;
  const double inv = rcp_nr(rb * s2);       // the one reciprocal: 1/(rho^2 B sin^2)
  const double irb = inv * s2;              // 1/(rho^2 B)
  p.R = irb * B;
  const double iB = irb * p.rho2;
  p.is2 = inv * rb;
  p.beta = twoMr * iB;
  p.h = p.rho2 * iB;
  p.zp1 = B * p.R;
  p.r2a2 = r2 + g.a2;
  p.r2 = r2;
  p.sc2 = (s + s) * c;
  return p;
}

// Right-hand sides X^i, U_i of Eq.(12) without the Lorentz force.
// epsz = eps (1+z): eps = 1 for massive particles, 0 for photons.
__device__ __forceinline__ void geodesic_rhs(const GridDev& g, const Pos& p, double epsz, double ur, double ut,
                                             double up, double& Xr, double& Xt, double& Xp,
                                             double& Ur, double& Ut) {
  const double R = p.R, R2 = R * R;
  const double ur2 = ur * ur, up2s = up * up * p.is2;
  const double aup = g.a * up;
  // P = rho^2 * (gamma^ij u_i u_j + beta u_r^2)
  const double P = fma(p.r2a2, ur2, fma(ut, ut, fma(2.0 * ur, aup, up2s)));
  const double N = fma(R, P, -p.beta * ur2);                 // gamma^ij u_i u_j
  const double G2 = fma(N, p.zp1, epsz);                     // (u^0)^2 = (eps+N)(1+z)
  const double iu0 = rsqrt_nr(G2);
  const double u0 = G2 * iu0;
  const double Riu0 = R * iu0;
  // gamma^{rj} u_j / u^0 - beta
  Xr = fma(fma(p.r2a2, ur, aup), Riu0, -p.beta * fma(ur, iu0, 1.0));
  Xt = Riu0 * ut;
  Xp = Riu0 * fma(up, p.is2, g.a * ur);
  // derivatives: dz/dr = 2M (a^2 c^2 - r^2)/rho^4, dz/dth = 4 M r a^2 s c / rho^4; W = 1/(1+z)^2;
  // a^2 c^2 - r^2 = rho^2 - 2 r^2
  const double A2 = g.a2 * p.sc2;                            // 2 a^2 sin cos
  const double WR2 = p.h * p.h * R2 * g.twoM;
  const double Wdzr = WR2 * fma(-2.0, p.r2, p.rho2);
  const double Wdzt = (WR2 * p.r) * A2;
  const double lead = fma(0.5, u0, ur);                      // (u^0/2 + u_r)
  // (d_i gamma^jk) u_j u_k
  const double twor = p.r + p.r;
  const double quad_r = fma(-twor * R2, P, (twor * R - Wdzr) * ur2);
  const double quad_t = fma(A2 * R2, P, -fma((R * p.is2) * p.sc2, up2s, Wdzt * ur2));
  const double hiu0 = 0.5 * iu0;
  Ur = fma(Wdzr, lead, -quad_r * hiu0);
  Ut = fma(Wdzt, lead, -quad_t * hiu0);
}

// Generalised Boris, full dt (Eq.16-19).  D, B contravariant.
__device__ __forceinline__ void boris(const GridDev& g, const Pos& p, double alpha, double sgn, double dt,
                                      const double D[3], const double B[3], double& ur, double& ut,
                                      double& up) {
  const double s2 = p.s * p.s;
  const double g_rr = p.zp1, g_tt = p.rho2;
  const double g_rp = -g.a * s2 * p.zp1;
  const double g_pp = s2 * fma(g.a2 * s2, p.zp1, p.rho2);
  const double sqrtg = p.rho2 * p.s * p.zp1 * alpha;
  const double gu_rr = fma(p.r2a2, p.R, -p.beta), gu_tt = p.R, gu_pp = p.R * p.is2, gu_rp = g.a * p.R;
  const double hdt = sgn * dt * 0.5;
  const double k = hdt * alpha;
  const double Dr = fma(g_rr, D[0], g_rp * D[2]), Dt = g_tt * D[1], Dp = fma(g_rp, D[0], g_pp * D[2]);
  const double mr = fma(k, Dr, ur), mt = fma(k, Dt, ut), mp = fma(k, Dp, up);   // u^-
  double ar = fma(gu_rr, mr, gu_rp * mp), at = gu_tt * mt, ap = fma(gu_rp, mr, gu_pp * mp);
  const double N = fma(ar, mr, fma(at, mt, ap * mp));
  const double f = hdt * alpha * rsqrt_nr(1.0 + N);                             // q dt / (2 ubar^0)
  const double tr = f * B[0], tt = f * B[1], tp = f * B[2];                     // t^i
  // u~ = u^- + sqrtg eps (u^-)^j t^k
  const double wr = fma(sqrtg, at * tp - ap * tt, mr);
  const double wt = fma(sqrtg, ap * tr - ar * tp, mt);
  const double wp = fma(sqrtg, ar * tt - at * tr, mp);
  const double t2 = fma(fma(g_rr, tr, g_rp * tp), tr, fma(g_tt * tt, tt, fma(g_rp, tr, g_pp * tp) * tp));
  const double sc = 2.0 * rcp_nr(1.0 + t2);
  const double sr = sc * tr, st = sc * tt, sp = sc * tp;
  ar = fma(gu_rr, wr, gu_rp * wp); at = gu_tt * wt; ap = fma(gu_rp, wr, gu_pp * wp);
  const double pr = fma(sqrtg, at * sp - ap * st, mr);                          // u^+
  const double pt = fma(sqrtg, ap * sr - ar * sp, mt);
  const double pp = fma(sqrtg, ar * st - at * sr, mp);
  ur = fma(k, Dr, pr); ut = fma(k, Dt, pt); up = fma(k, Dp, pp);
}

// Vay pusher in the FIDO frame (Vay 2008), full dt.  Orthonormal triad
// e_(1) = sqrt(gamma^rr)(d_r - gamma_rphi/gamma_phiphi d_phi), e_(2) = d_theta/sqrt(gamma_thth),
// e_(3) = d_phi/sqrt(gamma_phiphi); FIDO proper time alpha*dt.  D, B contravariant, u covariant.
__device__ __forceinline__ void vay(const GridDev& g, const Pos& p, double alpha, double sgn, double dt,
                                    const double D[3], const double B[3], double& ur, double& ut, double& up) {
  // square roots and quotients through the MUFU-seeded rsqrt_nr / rcp_nr (no division, no sqrt call)
  const double s2 = p.s * p.s;
  const double g_rp = -g.a * s2 * p.zp1, g_pp = s2 * fma(g.a2 * s2, p.zp1, p.rho2);
  const double gu_rr = fma(p.r2a2, p.R, -p.beta);
  const double isgrr = rsqrt_nr(gu_rr), isth = rsqrt_nr(p.rho2), isph = rsqrt_nr(g_pp);
  const double sgrr = gu_rr * isgrr, sth = p.rho2 * isth, sph = g_pp * isph;
  const double k = g_rp * (isph * isph);
  const double uh0 = sgrr * fma(-k, up, ur), uh1 = ut * isth, uh2 = up * isph;
  const double E0 = D[0] * isgrr, E1 = sth * D[1], E2 = fma(g_rp, D[0], g_pp * D[2]) * isph;
  const double B0 = B[0] * isgrr, B1 = sth * B[1], B2 = fma(g_rp, B[0], g_pp * B[2]) * isph;
  const double h = sgn * alpha * dt;
  const double iG0 = rsqrt_nr(fma(uh0, uh0, fma(uh1, uh1, fma(uh2, uh2, 1.0))));
  const double v0 = uh0 * iG0, v1 = uh1 * iG0, v2 = uh2 * iG0;
  const double p0 = fma(h, fma(0.5, v1 * B2 - v2 * B1, E0), uh0);
  const double p1 = fma(h, fma(0.5, v2 * B0 - v0 * B2, E1), uh1);
  const double p2 = fma(h, fma(0.5, v0 * B1 - v1 * B0, E2), uh2);
  const double hh = 0.5 * h;
  const double t0 = hh * B0, t1 = hh * B1, t2 = hh * B2;
  const double tau2 = fma(t0, t0, fma(t1, t1, t2 * t2));
  const double ustar = fma(p0, t0, fma(p1, t1, p2 * t2));
  const double sigma = fma(p0, p0, fma(p1, p1, fma(p2, p2, 1.0))) - tau2;
  const double disc = fma(sigma, sigma, 4.0 * fma(ustar, ustar, tau2));     // > 0: sigma >= 1 when tau = 0
  const double G12 = 0.5 * fma(disc, rsqrt_nr(disc), sigma);                // gamma_new^2
  const double iG1 = rsqrt_nr(G12);
  const double w0 = t0 * iG1, w1 = t1 * iG1, w2 = t2 * iG1;
  const double udt = fma(p0, w0, fma(p1, w1, p2 * w2));
  const double sc = rcp_nr(fma(w0, w0, fma(w1, w1, fma(w2, w2, 1.0))));
  const double n0 = sc * (fma(udt, w0, p0) + (p1 * w2 - p2 * w1));
  const double n1 = sc * (fma(udt, w1, p1) + (p2 * w0 - p0 * w2));
  const double n2 = sc * (fma(udt, w2, p2) + (p0 * w1 - p1 * w0));
  ur = fma(n0, isgrr, n2 * g_rp * isph);
  ut = sth * n1;
  up = sph * n2;
}

// F[...] += v unless v == 0: one DSETP + one predicated RED.E.ADD.F64 (no divergent branch, so
// no BSSY/BSYNC pair around every one of the 40 window slots).
__device__ __forceinline__ void red_add(double* p, double v) {
  asm volatile(
      "{ .reg .pred q; setp.neu.f64 q, %1, 0d0000000000000000; @q red.global.add.f64 [%0], %1; }" ::"l"(p),
      "d"(v)
      : "memory");
}
// Short series for steps |d| <= kSmallStep = 2^-8 (the dropped terms are < 1e-18 relative): the
// in-cell offset of a particle on grids of ~1000 cells and more, and dt X^theta <= dt / rho of every
// corrector at the production time steps.  Both share the four Taylor coefficients -1/6, 1/120,
// -1/24, 1/720.
constexpr double kSmallStep = 0.00390625;
// sin, cos of th0 + d from (s0, c0) by angle addition
__device__ __forceinline__ void sincos_shift(const PolyTab& pt, double s0, double c0, double d, double& s, double& c) {
  const double d2 = d * d;
  const double ps = fma(d2, pt.v[kR120], pt.v[kR6]);
  const double pc = fma(fma(d2, pt.v[kR720], pt.v[kR24]), d2, 0.5);
  const double sd = fma(ps * d2, d, d);                         // sin d
  const double vd = pc * d2;                                    // 1 - cos d
  s = s0 + fma(c0, sd, -s0 * vd);
  c = c0 - fma(s0, sd, c0 * vd);
}
// exp(d) - 1 = sinh d + (cosh d - 1): the same two polynomials evaluated at -d^2
__device__ __forceinline__ double expm1_small(const PolyTab& pt, double d) {
  const double m = -d * d;
  const double ps = fma(m, pt.v[kR120], pt.v[kR6]);
  const double pc = fma(fma(m, pt.v[kR720], pt.v[kR24]), m, 0.5);
  const double sh = fma(ps * m, d, d);                          // sinh d
  return fma(-pc, m, sh);                                       // + cosh d - 1
}

// General-window deposit (moves of more than one cell; never taken below the Courant limit).
__device__ __noinline__ void deposit_far(const GridDev* gp, double Q, double idt, double vphi,
                                         double xa, double xb, double ya, double yb, double* Fr,
                                         double* Fth, double* Fph, uint32_t* status) {
  const GridDev& g = *gp;
  const int ilo = (int)floor(fmin(xa, xb)), ihi = (int)floor(fmax(xa, xb)) + 1;
  const int jlo = (int)floor(fmin(ya, yb)), jhi = (int)floor(fmax(ya, yb)) + 1;
  if (status) atomicOr(status, GRPIC_STATUS_FAR_MOVE);
  if (ilo < -g.ng || ihi > g.nr + g.ng || jlo < -g.ng || jhi > g.nth + g.ng) {
    if (status) atomicOr(status, GRPIC_STATUS_OFFGRID);
    return;
  }
  auto S = [](double x) { return fmax(0.0, 1.0 - fabs(x)); };
  for (int j = jlo; j <= jhi; ++j) {
    double acc = 0.0;
    for (int i = ilo; i < ihi; ++i) {
      acc -= 0.5 * Q * (S(xb - i) - S(xa - i)) * (S(yb - j) + S(ya - j)) * idt;
      red_add(Fr + g.idx(i, j), acc);
    }
  }
  for (int i = ilo; i <= ihi; ++i) {
    double acc = 0.0;
    for (int j = jlo; j < jhi; ++j) {
      acc -= 0.5 * Q * (S(yb - j) - S(ya - j)) * (S(xb - i) + S(xa - i)) * idt;
      red_add(Fth + g.idx(i, j), acc);
    }
  }
  for (int j = jlo; j <= jhi; ++j)
    for (int i = ilo; i <= ihi; ++i)
      red_add(Fph + g.idx(i, j),
              vphi * ((1.0 / 3.0) * (S(xb - i) * S(yb - j) + S(xa - i) * S(ya - j)) +
                      (1.0 / 6.0) * (S(xb - i) * S(ya - j) + S(xa - i) * S(yb - j))));
}

}  // namespace
