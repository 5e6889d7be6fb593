// Fused GR particle push + charge-conserving current deposit (sm_100a).
//
// One thread per particle.  All Kerr-Schild metric terms (lapse, shift, spatial metric, inverse
// metric and the r/theta derivatives entering Eq.12) are computed inline in registers from
// (r, sin theta, cos theta); position-only terms are shared between the Boris rotation and
// the first geodesic right-hand side.  Closed forms: Appendix A with M
// restored; derivative forms are this file's own.
#include <math.h>

#include "grpic_internal.cuh"

namespace {

struct Pos {          // position-only terms at (r, theta)
  double r, s, c;     // r, sin, cos
  double R;           // 1/rho^2
  double is2;         // 1/sin^2
  double is;          // 1/sin
  double beta;        // beta^r = 2Mr/(rho^2+2Mr)
  double zp1;         // 1+z
  double h;           // 1/(1+z) = alpha^2
  double r2a2;        // r^2 + a^2
  double rho2;
};

__device__ __forceinline__ Pos make_pos(const GridDev& g, double r, double s, double c) {
  Pos p;
  p.r = r; p.s = s; p.c = c;
  p.rho2 = fma(g.a2 * c, c, r * r);
  const double twoMr = 2.0 * g.M * r;
  const double B = p.rho2 + twoMr;          // rho^2 (1+z)
  p.R = 1.0 / p.rho2;
  const double iB = 1.0 / B;
  p.is = 1.0 / s;
  p.is2 = p.is * p.is;
  p.beta = twoMr * iB;
  p.h = p.rho2 * iB;
  p.zp1 = B * p.R;
  p.r2a2 = fma(r, r, g.a2);
  return p;
}

// Right-hand sides X^i, U_i of Eq.(12) without the Lorentz force.
__device__ __forceinline__ void geodesic_rhs(const GridDev& g, const Pos& p, double ur, double ut,
                                             double up, double& Xr, double& Xt, double& Xp,
                                             double& Ur, double& Ut) {
  const double R = p.R, R2 = R * R;
  const double ur2 = ur * ur, up2s = up * up * p.is2;
  // P = rho^2 * (gamma^ij u_i u_j + beta u_r^2)
  const double P = fma(p.r2a2, ur2, fma(ut, ut, fma(2.0 * g.a * ur, up, up2s)));
  const double N = fma(R, P, -p.beta * ur2);                 // gamma^ij u_i u_j
  const double G2 = (1.0 + N) * p.zp1;                       // (u^0)^2
  const double iu0 = rsqrt(G2);
  const double u0 = G2 * iu0;
  const double gur = fma(p.r2a2 * R - p.beta, ur, g.a * R * up);   // gamma^{rj} u_j
  Xr = fma(gur, iu0, -p.beta);
  Xt = R * ut * iu0;
  Xp = R * fma(up, p.is2, g.a * ur) * iu0;
  // derivatives: dz/dr = 2M (a^2 c^2 - r^2)/rho^4, dz/dth = 4 M r a^2 s c / rho^4
  const double A = g.a2 * p.s * p.c;
  const double W = p.h * p.h;
  const double Wdzr = W * 2.0 * g.M * (g.a2 * p.c * p.c - p.r * p.r) * R2;
  const double Wdzt = W * 4.0 * g.M * p.r * A * R2;
  const double lead = fma(0.5, u0, ur);                      // (u^0/2 + u_r)
  // (d_i gamma^jk) u_j u_k
  const double quad_r = fma(-2.0 * p.r * R2, P, fma(2.0 * p.r * R, ur2, -Wdzr * ur2));
  const double quad_t = fma(2.0 * A * R2, P, fma(-2.0 * R * p.c * p.is, up2s, -Wdzt * ur2));
  const double hiu0 = 0.5 * iu0;
  Ur = fma(Wdzr, lead, -quad_r * hiu0);
  Ut = fma(Wdzt, lead, -quad_t * hiu0);
}

// Generalised Boris, full dt (Eq.16-19).  D, B contravariant.
__device__ __forceinline__ void boris(const GridDev& g, const Pos& p, double sgn, double dt,
                                      const double D[3], const double B[3], double& ur, double& ut,
                                      double& up) {
  const double s2 = p.s * p.s;
  const double g_rr = p.zp1, g_tt = p.rho2;
  const double g_rp = -g.a * s2 * p.zp1;
  const double g_pp = s2 * fma(g.a2 * s2, p.zp1, p.rho2);
  const double alpha = sqrt(p.h);
  const double sqrtg = p.rho2 * p.s * p.zp1 * alpha;
  const double gu_rr = p.r2a2 * p.R - p.beta, gu_tt = p.R, gu_pp = p.R * p.is2, gu_rp = g.a * p.R;
  const double k = sgn * alpha * dt * 0.5;
  const double Dr = fma(g_rr, D[0], g_rp * D[2]), Dt = g_tt * D[1], Dp = fma(g_rp, D[0], g_pp * D[2]);
  const double mr = fma(k, Dr, ur), mt = fma(k, Dt, ut), mp = fma(k, Dp, up);   // u^-
  const double N = fma(gu_rr * mr, mr, fma(gu_tt * mt, mt, fma(gu_pp * mp, mp, 2.0 * gu_rp * mr * mp)));
  const double iu0 = alpha * rsqrt(1.0 + N);                                    // 1/ubar^0
  const double f = sgn * dt * 0.5 * iu0;
  const double tr = f * B[0], tt = f * B[1], tp = f * B[2];                     // t^i
  // u~ = u^- + sqrtg eps (u^-)^j t^k
  double ar = fma(gu_rr, mr, gu_rp * mp), at = gu_tt * mt, ap = fma(gu_rp, mr, gu_pp * mp);
  const double wr = fma(sqrtg, at * tp - ap * tt, mr);
  const double wt = fma(sqrtg, ap * tr - ar * tp, mt);
  const double wp = fma(sqrtg, ar * tt - at * tr, mp);
  const double t2 = fma(fma(g_rr, tr, g_rp * tp), tr, fma(g_tt * tt, tt, fma(g_rp, tr, g_pp * tp) * tp));
  const double sc = 2.0 / (1.0 + t2);
  const double sr = sc * tr, st = sc * tt, sp = sc * tp;
  ar = fma(gu_rr, wr, gu_rp * wp); at = gu_tt * wt; ap = fma(gu_rp, wr, gu_pp * wp);
  const double pr = fma(sqrtg, at * sp - ap * st, mr);                          // u^+
  const double pt = fma(sqrtg, ap * sr - ar * sp, mt);
  const double pp = fma(sqrtg, ar * st - at * sr, mp);
  ur = fma(k, Dr, pr); ut = fma(k, Dt, pt); up = fma(k, Dp, pp);
}

__device__ __forceinline__ double bilin(const double* __restrict__ F, size_t base, int pitch,
                                        double wx, double wy) {
  const double f00 = __ldg(F + base), f10 = __ldg(F + base + 1);
  const double f01 = __ldg(F + base + pitch), f11 = __ldg(F + base + pitch + 1);
  const double lo = fma(wx, f10 - f00, f00), hi = fma(wx, f11 - f01, f01);
  return fma(wy, hi - lo, lo);
}

__device__ __forceinline__ void red_add(double* p, double v) {
  if (v != 0.0) atomicAdd(p, v);   // result unused -> RED.E.ADD.F64
}

// General-window deposit (moves of more than one cell; never taken below the Courant limit).
__device__ __noinline__ void deposit_far(const GridDev& g, double Q, double idt, double vphi,
                                         double xa, double xb, double ya, double yb, double* Fr,
                                         double* Fth, double* Fph, uint32_t* status) {
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

__device__ __forceinline__ void shape3(double d, double S[3]) {
  // CIC weights of a point at offset d in [0,2) from the first of three consecutive nodes
  S[0] = fmax(0.0, 1.0 - d);
  S[1] = 1.0 - fabs(d - 1.0);
  S[2] = fmax(0.0, d - 1.0);
}

__global__ void __launch_bounds__(128)
push_deposit_kernel(GridDev g, grpic_particles ptc, grpic_fields f, grpic_current J, double dt,
                    int K, uint32_t* status) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= ptc.n) return;
  const uint32_t flag = ptc.flag[k];
  if (flag & 2u) return;
  const double x1 = ptc.x1[k], x2 = ptc.x2[k], x3 = ptc.x3[k];
  double ur = ptc.u1[k], ut = ptc.u2[k], up = ptc.u3[k];
  const double w = ptc.w[k];
  const double sgn = (flag & 1u) ? 1.0 : -1.0;

  // ---- gather (first order, each component from its own staggered lattice) ----
  const double xa = (x1 - g.xi_in) * g.inv_dxi, ya = x2 * g.inv_dth;
  double D[3], B[3];
  {
    const double fin = floor(xa), fjn = floor(ya);
    const double fih = floor(xa - 0.5), fjh = floor(ya - 0.5);
    const int in = (int)fin, jn = (int)fjn, ih = (int)fih, jh = (int)fjh;
    const double wxn = xa - fin, wyn = ya - fjn, wxh = xa - 0.5 - fih, wyh = ya - 0.5 - fjh;
    D[0] = bilin(f.Dr, g.idx(ih, jn), g.pitch, wxh, wyn);
    D[1] = bilin(f.Dth, g.idx(in, jh), g.pitch, wxn, wyh);
    D[2] = bilin(f.Dph, g.idx(in, jn), g.pitch, wxn, wyn);
    B[0] = bilin(f.Br, g.idx(in, jh), g.pitch, wxn, wyh);
    B[1] = bilin(f.Bth, g.idx(ih, jn), g.pitch, wxh, wyn);
    B[2] = bilin(f.Bph, g.idx(ih, jh), g.pitch, wxh, wyh);
  }

  // ---- Boris (full dt) at x^n ----
  const double r0 = exp(x1);
  double s, c;
  sincos(x2, &s, &c);
  const Pos p0 = make_pos(g, r0, s, c);
  boris(g, p0, sgn, dt, D, B, ur, ut, up);

  // ---- geodesic predictor + K correctors (Eq.14, 15) ----
  double Xr0, Xt0, Xp0, Ur0, Ut0;
  geodesic_rhs(g, p0, ur, ut, up, Xr0, Xt0, Xp0, Ur0, Ut0);
  double r = fma(Xr0, dt, r0), th = fma(Xt0, dt, x2), ph = fma(Xp0, dt, x3);
  double vr = fma(Ur0, dt, ur), vt = fma(Ut0, dt, ut);
  const double hdt = 0.5 * dt;
  for (int it = 0; it < K; ++it) {
    sincos(th, &s, &c);
    const Pos p1 = make_pos(g, r, s, c);
    double Xr, Xt, Xp, Ur, Ut;
    geodesic_rhs(g, p1, vr, vt, up, Xr, Xt, Xp, Ur, Ut);
    r = fma(hdt, Xr + Xr0, r0);
    th = fma(hdt, Xt + Xt0, x2);
    ph = fma(hdt, Xp + Xp0, x3);
    vr = fma(hdt, Ur + Ur0, ur);
    vt = fma(hdt, Ut + Ut0, ut);
  }

  // ---- new logical position, reflection, removal ----
  const double x1n = log(r);
  const double th_dep = th;
  if (th < 0.0) { th = -th; vt = -vt; }
  if (th > M_PI) { th = 2.0 * M_PI - th; vt = -vt; }
  uint32_t nflag = flag, ncell;
  const bool finite = isfinite(x1n) && isfinite(th) && isfinite(ph) && isfinite(vr) && isfinite(vt);
  const bool out = !finite || (x1n < g.xi_in) || (x1n >= g.xi_out);
  if (out) {
    nflag |= 2u;
    ncell = 0xFFFFFFFFu;
    if (!finite && status) atomicOr(status, GRPIC_STATUS_NONFINITE);
  } else {
    int ic = (int)floor((x1n - g.xi_in) / g.dxi);
    int jc = (int)floor(th / g.dth);
    ic = min(max(ic, 0), g.nr - 1);
    jc = min(max(jc, 0), g.nth - 1);
    ncell = (uint32_t)(jc * g.nr + ic);
  }
  ptc.x1[k] = x1n; ptc.x2[k] = th; ptc.x3[k] = ph;
  ptc.u1[k] = vr; ptc.u2[k] = vt; ptc.u3[k] = up;
  ptc.cell[k] = ncell;
  ptc.flag[k] = nflag;
  if (!finite) return;

  // ---- charge-conserving deposit of the move (Eq.21-23) ----
  const double xb = (x1n - g.xi_in) * g.inv_dxi, yb = th_dep * g.inv_dth;
  const double Q = sgn * w, idt = 1.0 / dt;
  const double vphi = Q * (ph - x3) * idt;
  const int ia = (int)floor(xa), ib = (int)floor(xb), ja = (int)floor(ya), jb = (int)floor(yb);
  const int i0 = min(ia, ib), j0 = min(ja, jb);
  if (max(ia, ib) - i0 > 1 || max(ja, jb) - j0 > 1) {
    deposit_far(g, Q, idt, vphi, xa, xb, ya, yb, J.Fr, J.Fth, J.Fph, status);
    return;
  }
  if (i0 < -g.ng || i0 + 2 > g.nr + g.ng || j0 < -g.ng || j0 + 2 > g.nth + g.ng) {
    if (status) atomicOr(status, GRPIC_STATUS_OFFGRID);
    return;
  }
  double Sa[3], Sb[3], Ta[3], Tb[3];
  shape3(xa - i0, Sa); shape3(xb - i0, Sb); shape3(ya - j0, Ta); shape3(yb - j0, Tb);
  const size_t base = g.idx(i0, j0);
  const double hq = -0.5 * Q * idt;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    const double at = hq * (Tb[j] + Ta[j]);
    const double f0 = at * (Sb[0] - Sa[0]);                 // F_r(i0+1/2, j0+j)
    const double f1 = fma(at, Sb[1] - Sa[1], f0);           // F_r(i0+3/2, j0+j)
    red_add(J.Fr + base + (size_t)j * g.pitch, f0);
    red_add(J.Fr + base + (size_t)j * g.pitch + 1, f1);
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const double as = hq * (Sb[i] + Sa[i]);
    const double f0 = as * (Tb[0] - Ta[0]);                 // F_th(i0+i, j0+1/2)
    const double f1 = fma(as, Tb[1] - Ta[1], f0);           // F_th(i0+i, j0+3/2)
    red_add(J.Fth + base + i, f0);
    red_add(J.Fth + base + g.pitch + i, f1);
  }
#pragma unroll
  for (int j = 0; j < 3; ++j)
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const double sh = (1.0 / 3.0) * fma(Sb[i], Tb[j], Sa[i] * Ta[j]) +
                        (1.0 / 6.0) * fma(Sb[i], Ta[j], Sa[i] * Tb[j]);
      red_add(J.Fph + base + (size_t)j * g.pitch + i, vphi * sh);
    }
}

}  // namespace

extern "C" int grpic_push_deposit(grpic_ctx* ctx, grpic_particles* ptc, const grpic_fields* fields,
                                  grpic_current* flux, double dt, uint32_t* status, void* stream) {
  if (!ctx || !ptc || !fields || !flux || !(dt > 0.0) || ptc->n < 0) return GRPIC_ERR_ARG;
  if (!ptc->x1 || !ptc->x2 || !ptc->x3 || !ptc->u1 || !ptc->u2 || !ptc->u3 || !ptc->w ||
      !ptc->cell || !ptc->flag)
    return GRPIC_ERR_ARG;
  if (!fields->Dr || !fields->Dth || !fields->Dph || !fields->Br || !fields->Bth || !fields->Bph ||
      !flux->Fr || !flux->Fth || !flux->Fph)
    return GRPIC_ERR_ARG;
  if (ptc->n == 0) return GRPIC_OK;
  const int block = 128;
  const int64_t grid = (ptc->n + block - 1) / block;
  if (grid > 0x7FFFFFFFLL) return GRPIC_ERR_ARG;
  push_deposit_kernel<<<(unsigned)grid, block, 0, (cudaStream_t)stream>>>(
      ctx->g, *ptc, *fields, *flux, dt, ctx->p.geo_iters, status);
  grpic_count_launches(1);
  return grpic_launch_ok();
}
