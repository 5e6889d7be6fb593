// The paper's method VARIANTS of the particle step (general kernel, one thread per particle; the tuned
// first-order / Boris default lives in push_deposit.cu, which also takes first-order / Vay):
//  * shape order 3: the THIRD-ORDER (cubic B-spline) particle shape, the paper's configuration
//    option: field gather over the 4 x 4 nodes of the spline's support on each
//    component's own staggered lattice, prefix-sum deposit (Eq.21-23) over the window the spline
//    covers during the move (5 x 5 nodes for a move of less than one cell); order 1 = cloud-in-cell;
//  * pusher 1: the Vay momentum update in the FIDO frame instead of the generalised
//    Boris update; the geodesic part is the same.
#include <math.h>

#include "grpic_internal.cuh"
#include "push_math.cuh"

namespace {

// ORDER 3: cubic B-spline 2/3 - x^2 + |x|^3/2 (|x| < 1), (2 - |x|)^3/6 (1 <= |x| < 2), 0 beyond;
// ORDER 1: cloud-in-cell max(0, 1 - |x|)
template <int ORDER>
__device__ __forceinline__ double shp(double x) {
  const double ax = fabs(x);
  if (ORDER == 1) return ax < 1.0 ? 1.0 - ax : 0.0;
  // both pieces are evaluated and selected (no branch: 4 (4 + 2 EXT) calls per particle in the deposit)
  const double inner = fma(ax * ax, fma(0.5, ax, -1.0), 2.0 / 3.0);
  const double t = 2.0 - ax;
  const double outer = t * t * t * (1.0 / 6.0);
  return ax < 1.0 ? inner : (ax < 2.0 ? outer : 0.0);
}

// F[...] += v if ok and v != 0: predicated RED, no branch
__device__ __forceinline__ void red_add_if(double* p, double v, bool ok) {
  asm volatile(
      "{ .reg .pred q, o; setp.ne.s32 o, %2, 0; setp.neu.and.f64 q, %1, 0d0000000000000000, o;\n"
      "@q red.global.add.f64 [%0], %1; }" ::"l"(p),
      "d"(v), "r"((int)ok)
      : "memory");
}

// the four (ORDER 3) / two (ORDER 1) non-zero weights of the nodes i0 .. i0 + 3, i0 = floor(gx) - 1, from
// the in-cell fraction fr = gx - floor(gx): distances 1 + fr, fr, 1 - fr, 2 - fr
template <int ORDER>
__device__ __forceinline__ void weights4(double fr, double w[4]) {
  const double g1 = 1.0 - fr;
  if (ORDER == 1) { w[0] = 0.0; w[1] = g1; w[2] = fr; w[3] = 0.0; return; }
  w[0] = g1 * g1 * g1 * (1.0 / 6.0);
  w[1] = fma(fr * fr, fma(0.5, fr, -1.0), 2.0 / 3.0);
  w[2] = fma(g1 * g1, fma(0.5, g1, -1.0), 2.0 / 3.0);
  w[3] = fr * fr * fr * (1.0 / 6.0);
}

// values of NC staggered components that share one lattice at logical position (gx, gy): sum over the
// 4 x 4 nodes around it (ORDER 1: the inner 2 x 2).  The weights are formed once per lattice and the
// loads of all NC components are issued before the first sum (the gather is latency-bound: 96 loads per
// particle at ORDER 3).
template <int ORDER, int NC>
__device__ __forceinline__ void gather_s(const GridDev& g, const double* const (&F)[NC], double gx, double gy,
                                         double (&out)[NC]) {
  const double fi = floor(gx), fj = floor(gy);
  const int i0 = (int)fi - 1, j0 = (int)fj - 1;
  double wx[4], wy[4];
  weights4<ORDER>(gx - fi, wx);
  weights4<ORDER>(gy - fj, wy);
  constexpr int LO = ORDER == 1 ? 1 : 0, HI = ORDER == 1 ? 3 : 4;
  const size_t base = g.idx(i0, j0);
  double v[NC][4][4];
#pragma unroll
  for (int c = 0; c < NC; ++c)
#pragma unroll
    for (int n = LO; n < HI; ++n)
#pragma unroll
      for (int m = LO; m < HI; ++m) v[c][n][m] = __ldg(F[c] + base + (size_t)n * g.pitch + m);
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    double acc = 0.0;
#pragma unroll
    for (int n = LO; n < HI; ++n) {
      double r = 0.0;
#pragma unroll
      for (int m = LO; m < HI; ++m) r = fma(wx[m], v[c][n][m], r);
      acc = fma(wy[n], r, acc);
    }
    out[c] = acc;
  }
}

// resident 128-thread CTAs per SM asked of the compiler (register cap 65536 / (128 MINB)).  The kernel
// waits on its gather loads (long scoreboard): more warps help more than the spills cost.  Cubic shape at
// 2e7 particles, ms per push: 1 (128 registers): 5.89, 5 (96, 40 B of stack): 5.07, 6 (80): 5.09, 8 (64): 5.30
#ifndef GRPIC_S3_MINB
#define GRPIC_S3_MINB 5
#endif
template <int ORDER>
__global__ void __launch_bounds__(128, GRPIC_S3_MINB)
push_deposit_general_kernel(const __grid_constant__ GridDev g, const __grid_constant__ grpic_particles ptc,
                            const __grid_constant__ grpic_fields f, const __grid_constant__ grpic_current J,
                            const __grid_constant__ PolyTab pt, double dt, int K, int pusher, uint32_t* status) {
  constexpr int EXT = ORDER == 3 ? 1 : 0;            // extra nodes of support on each side
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= ptc.n) return;
  // the whole particle is requested at once (round trips to HBM one after the other otherwise: flag, then
  // the position, then -- behind the gather -- the momentum, phi and the weight)
  const uint32_t flag = ptc.flag[k];
  const double x1 = ptc.x1[k], x2 = ptc.x2[k], x3 = ptc.x3[k];
  const double u1 = ptc.u1[k], u2 = ptc.u2[k], u3 = ptc.u3[k], wgt = ptc.w[k];
  if (flag & 2u) return;
  const bool photon = (flag & 4u) != 0;
  const double sgn = photon ? 0.0 : ((flag & 1u) ? 1.0 : -1.0);
  const double idt = 1.0 / dt;
  const double xa = (x1 - g.xi_in) * g.inv_dxi, ya = x2 * g.inv_dth;

  // ---- gather: D^r,B^th at (i+1/2, j); D^th,B^r at (i, j+1/2); D^ph at (i, j); B^ph at (i+1/2, j+1/2)
  double D[3] = {0.0, 0.0, 0.0}, B[3] = {0.0, 0.0, 0.0};
  if (!photon) {
    double o2[2], o1[1];
    { const double* const F2[2] = {f.Dr, f.Bth}; gather_s<ORDER, 2>(g, F2, xa - 0.5, ya, o2); D[0] = o2[0]; B[1] = o2[1]; }
    { const double* const F2[2] = {f.Dth, f.Br}; gather_s<ORDER, 2>(g, F2, xa, ya - 0.5, o2); D[1] = o2[0]; B[0] = o2[1]; }
    { const double* const F1[1] = {f.Dph}; gather_s<ORDER, 1>(g, F1, xa, ya, o1); D[2] = o1[0]; }
    { const double* const F1[1] = {f.Bph}; gather_s<ORDER, 1>(g, F1, xa - 0.5, ya - 0.5, o1); B[2] = o1[0]; }
  }

  // ---- Boris / Vay (full dt) at x^n, then geodesic predictor + K correctors (Eq.14, 15); exp, sincos and
  // ln r are the kernel's own (push_math.cuh), with the short series where the step allows them ----
  const double r0 = exp_pt(pt, x1);
  double s0, c0;
  sincos_pt(pt, x2, s0, c0);
  const Pos p0 = make_pos(g, r0, s0, c0);
  const double alpha0 = p0.h * rsqrt_nr(p0.h);
  double ur = u1, ut = u2, up = u3;
  if (pusher == 1) vay(g, p0, alpha0, sgn, dt, D, B, ur, ut, up);
  else boris(g, p0, alpha0, sgn, dt, D, B, ur, ut, up);
  double Xr0, Xt0, Xp0, Ur0, Ut0;
  geodesic_rhs(g, p0, photon ? 0.0 : p0.zp1, ur, ut, up, Xr0, Xt0, Xp0, Ur0, Ut0);
  double dr = Xr0 * dt, dth = Xt0 * dt, dph = Xp0 * dt;
  double vr = fma(Ur0, dt, ur), vt = fma(Ut0, dt, ut);
  const double hdt = 0.5 * dt;
  for (int ci = 0; ci < K; ++ci) {
    double s, c;
    if (fabs(dth) <= kSmallStep) sincos_shift(pt, s0, c0, dth, s, c);
    else sincos_pt(pt, x2 + dth, s, c);
    const Pos p1 = make_pos(g, r0 + dr, s, c);
    double Xr, Xt, Xp, Ur, Ut;
    geodesic_rhs(g, p1, photon ? 0.0 : p1.zp1, vr, vt, up, Xr, Xt, Xp, Ur, Ut);
    dr = hdt * (Xr + Xr0);
    dth = hdt * (Xt + Xt0);
    dph = hdt * (Xp + Xp0);
    vr = fma(hdt, Ur + Ur0, ur);
    vt = fma(hdt, Ut + Ut0, ut);
  }
  // ln r = x1 + 2 atanh(dr / (2 r0 + dr))
  double x1n;
  {
    const double wq = dr * rcp_nr(r0 + (r0 + dr));
    if (fabs(wq) <= 0.03) {
      const double w2 = wq * wq;
      double pl = fma(w2, pt.v[kR11], pt.v[kR9]);
      pl = fma(pl, w2, pt.v[kR7]);
      pl = fma(pl, w2, pt.v[kR5]);
      pl = fma(pl, w2, pt.v[kR3]);
      x1n = fma(2.0, fma(pl * w2, wq, wq), x1);
    } else {
      x1n = log(r0 + dr);
    }
  }
  const double ph = x3 + dph;
  double th = x2 + dth;
  const double th_dep = th;
  if (th < 0.0) { th = -th; vt = -vt; }
  if (th > M_PI) { th = 2.0 * M_PI - th; vt = -vt; }

  // ---- removal flag, new cell (floor of the quotient, as in push_deposit.cu) ----
  uint32_t nflag = flag, ncell;
  const bool finite = isfinite(x1n) && isfinite(th) && isfinite(ph) && isfinite(vr) && isfinite(vt);
  if (!finite || x1n < g.xi_in || x1n >= g.xi_out) {
    nflag |= 2u;
    ncell = 0xFFFFFFFFu;
    if (!finite && status) atomicOr(status, GRPIC_STATUS_NONFINITE);
  } else {
    int ic = (int)floor((x1n - g.xi_in) / g.dxi), jc = (int)floor(th / g.dth);
    ic = min(max(ic, 0), g.nr - 1);
    jc = min(max(jc, 0), g.nth - 1);
    ncell = (uint32_t)(jc * g.nr + ic);
  }
  ptc.x1[k] = x1n; ptc.x2[k] = th; ptc.x3[k] = ph;
  ptc.u1[k] = vr; ptc.u2[k] = vt; ptc.u3[k] = up;
  ptc.cell[k] = ncell;
  ptc.flag[k] = nflag;
  if (!finite || photon) return;

  // ---- deposit on the window the spline covers during the move (Eq.21-23) ----
  const double Q = sgn * wgt, vphi = Q * dph * idt;
  const double xb = (x1n - g.xi_in) * g.inv_dxi, yb = th_dep * g.inv_dth;
  const int ilo = (int)floor(fmin(xa, xb)) - EXT, ihi = (int)floor(fmax(xa, xb)) + 1 + EXT;
  const int jlo = (int)floor(fmin(ya, yb)) - EXT, jhi = (int)floor(fmax(ya, yb)) + 1 + EXT;
  constexpr int W = 4 + 2 * EXT;                    // nodes per direction of a move of less than one cell
  const int wi = ihi - ilo, wj = jhi - jlo;          // faces per direction (nodes - 1)
  if (wi > W - 1 || wj > W - 1) { if (status) atomicOr(status, GRPIC_STATUS_FAR_MOVE); }
  if (ilo < -g.ng || ihi > g.nr + g.ng || jlo < -g.ng || jhi > g.nth + g.ng) {
    if (status) atomicOr(status, GRPIC_STATUS_OFFGRID);
    return;
  }
  if (wi <= W - 1 && wj <= W - 1) {
    // the usual case: the shapes of the old and new position on the window's nodes are evaluated once
    // (4 W values instead of one per flux slot), the loops have compile-time bounds
    double Sa[W], Sb[W], Ta[W], Tb[W];
#pragma unroll
    for (int m = 0; m < W; ++m) {
      Sa[m] = shp<ORDER>(xa - (double)(ilo + m)); Sb[m] = shp<ORDER>(xb - (double)(ilo + m));
      Ta[m] = shp<ORDER>(ya - (double)(jlo + m)); Tb[m] = shp<ORDER>(yb - (double)(jlo + m));
    }
    const double hq = -0.5 * Q * idt;
    double* const fr = J.Fr + g.idx(ilo, jlo);
    double* const ft = J.Fth + g.idx(ilo, jlo);
    double* const fp = J.Fph + g.idx(ilo, jlo);
#pragma unroll
    for (int n = 0; n < W; ++n) {                    // F_r: W rows of W - 1 faces
      const double ty = hq * (Tb[n] + Ta[n]);
      double acc = 0.0;
#pragma unroll
      for (int m = 0; m < W - 1; ++m) {
        acc = fma(ty, Sb[m] - Sa[m], acc);
        red_add_if(fr + n * g.pitch + m, acc, n <= wj && m < wi);
      }
    }
#pragma unroll
    for (int m = 0; m < W; ++m) {                    // F_theta: W columns of W - 1 faces
      const double tx = hq * (Sb[m] + Sa[m]);
      double acc = 0.0;
#pragma unroll
      for (int n = 0; n < W - 1; ++n) {
        acc = fma(tx, Tb[n] - Ta[n], acc);
        red_add_if(ft + n * g.pitch + m, acc, m <= wi && n < wj);
      }
    }
#pragma unroll
    for (int n = 0; n < W; ++n) {                    // F_phi: W x W nodes
      const double U = vphi * fma(1.0 / 3.0, Tb[n], (1.0 / 6.0) * Ta[n]), V = vphi * fma(1.0 / 3.0, Ta[n], (1.0 / 6.0) * Tb[n]);
#pragma unroll
      for (int m = 0; m < W; ++m) red_add_if(fp + n * g.pitch + m, fma(Sb[m], U, Sa[m] * V), n <= wj && m <= wi);
    }
    return;
  }
  for (int j = jlo; j <= jhi; ++j) {
    const double ty = -0.5 * Q * idt * (shp<ORDER>(yb - j) + shp<ORDER>(ya - j));
    double acc = 0.0;
    for (int i = ilo; i < ihi; ++i) {
      acc = fma(ty, shp<ORDER>(xb - i) - shp<ORDER>(xa - i), acc);
      red_add(J.Fr + g.idx(i, j), acc);
    }
  }
  for (int i = ilo; i <= ihi; ++i) {
    const double tx = -0.5 * Q * idt * (shp<ORDER>(xb - i) + shp<ORDER>(xa - i));
    double acc = 0.0;
    for (int j = jlo; j < jhi; ++j) {
      acc = fma(tx, shp<ORDER>(yb - j) - shp<ORDER>(ya - j), acc);
      red_add(J.Fth + g.idx(i, j), acc);
    }
  }
  for (int j = jlo; j <= jhi; ++j) {
    const double Tb = shp<ORDER>(yb - j), Ta = shp<ORDER>(ya - j);
    const double U = vphi * fma(1.0 / 3.0, Tb, (1.0 / 6.0) * Ta), V = vphi * fma(1.0 / 3.0, Ta, (1.0 / 6.0) * Tb);
    for (int i = ilo; i <= ihi; ++i) red_add(J.Fph + g.idx(i, j), fma(shp<ORDER>(xb - i), U, shp<ORDER>(xa - i) * V));
  }
}

}  // namespace

extern "C" int grpic_push_deposit_variant(grpic_ctx* ctx, grpic_particles* ptc, const grpic_fields* fields,
                                          grpic_current* flux, double dt, int32_t shape_order, int32_t pusher,
                                          uint32_t* status, void* stream) {
  if (!ctx || !ptc || !fields || !flux || !(dt > 0.0) || ptc->n < 0) return GRPIC_ERR_ARG;
  if ((shape_order != 1 && shape_order != 3) || (pusher != 0 && pusher != 1)) return GRPIC_ERR_ARG;
  if (shape_order == 3 && ctx->g.ng < 3) return GRPIC_ERR_ARG;   // the spline's support needs three guard nodes
  if (ptc->n == 0) return GRPIC_OK;
  if (!ptc->x1 || !ptc->x2 || !ptc->x3 || !ptc->u1 || !ptc->u2 || !ptc->u3 || !ptc->w || !ptc->cell ||
      !ptc->flag || !fields->Dr || !fields->Dth || !fields->Dph || !fields->Br || !fields->Bth ||
      !fields->Bph || !flux->Fr || !flux->Fth || !flux->Fph)
    return GRPIC_ERR_ARG;
  const int64_t grid = (ptc->n + 127) / 128;
  if (grid > 0x7FFFFFFFLL) return GRPIC_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  if (shape_order == 1 && pusher == 1) {
    // first-order shape + Vay: the tuned kernel of push_deposit.cu with the Vay update in place of Boris
    const int rc = grpic_push_deposit_cic_vay(ctx, ptc, fields, flux, dt, status, st);
    if (rc != GRPIC_ERR_ARG) return rc;               // arrays off the 16-byte grid: the general kernel below
  }
  if (shape_order == 3)
    push_deposit_general_kernel<3><<<(unsigned)grid, 128, 0, st>>>(ctx->g, *ptc, *fields, *flux, kPolyTabHost, dt,
                                                                   ctx->p.geo_iters, pusher, status);
  else
    push_deposit_general_kernel<1><<<(unsigned)grid, 128, 0, st>>>(ctx->g, *ptc, *fields, *flux, kPolyTabHost, dt,
                                                                   ctx->p.geo_iters, pusher, status);
  grpic_count_launches(1);
  return grpic_launch_ok();
}

extern "C" int grpic_push_deposit_spline3(grpic_ctx* ctx, grpic_particles* ptc, const grpic_fields* fields,
                                          grpic_current* flux, double dt, uint32_t* status, void* stream) {
  return grpic_push_deposit_variant(ctx, ptc, fields, flux, dt, 3, 0, status, stream);
}
