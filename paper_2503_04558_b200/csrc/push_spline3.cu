// The paper's method VARIANTS of the particle step (general kernel, one thread per particle,
// straightforward loops; built for parity, not tuned -- the tuned default lives in push_deposit.cu):
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
  if (ax < 1.0) return fma(ax * ax, fma(0.5, ax, -1.0), 2.0 / 3.0);
  if (ax < 2.0) { const double t = 2.0 - ax; return t * t * t * (1.0 / 6.0); }
  return 0.0;
}

// value of one staggered component at logical position (gx, gy): sum over the 4 x 4 nodes around
// it (for ORDER 1 the outer ring has zero weight)
template <int ORDER>
__device__ __forceinline__ double gather_s(const GridDev& g, const double* __restrict__ F, double gx,
                                           double gy) {
  const double fi = floor(gx), fj = floor(gy);
  const int i0 = (int)fi - 1, j0 = (int)fj - 1;
  double wx[4], wy[4];
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    wx[m] = shp<ORDER>(gx - (double)(i0 + m));
    wy[m] = shp<ORDER>(gy - (double)(j0 + m));
  }
  double acc = 0.0;
#pragma unroll
  for (int n = 0; n < 4; ++n) {
    const double* row = F + g.idx(i0, j0 + n);
    double r = 0.0;
#pragma unroll
    for (int m = 0; m < 4; ++m) r = fma(wx[m], __ldg(row + m), r);
    acc = fma(wy[n], r, acc);
  }
  return acc;
}

template <int ORDER>
__global__ void __launch_bounds__(128)
push_deposit_general_kernel(const __grid_constant__ GridDev g, const __grid_constant__ grpic_particles ptc,
                            const __grid_constant__ grpic_fields f, const __grid_constant__ grpic_current J,
                            double dt, int K, int pusher, uint32_t* status) {
  constexpr int EXT = ORDER == 3 ? 1 : 0;            // extra nodes of support on each side
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= ptc.n) return;
  const uint32_t flag = ptc.flag[k];
  if (flag & 2u) return;
  const double x1 = ptc.x1[k], x2 = ptc.x2[k];
  const bool photon = (flag & 4u) != 0;
  const double sgn = photon ? 0.0 : ((flag & 1u) ? 1.0 : -1.0);
  const double idt = 1.0 / dt;
  const double xa = (x1 - g.xi_in) * g.inv_dxi, ya = x2 * g.inv_dth;

  // ---- gather: D^r,B^th at (i+1/2, j); D^th,B^r at (i, j+1/2); D^ph at (i, j); B^ph at (i+1/2, j+1/2)
  double D[3] = {0.0, 0.0, 0.0}, B[3] = {0.0, 0.0, 0.0};
  if (!photon) {
    D[0] = gather_s<ORDER>(g, f.Dr, xa - 0.5, ya);
    D[1] = gather_s<ORDER>(g, f.Dth, xa, ya - 0.5);
    D[2] = gather_s<ORDER>(g, f.Dph, xa, ya);
    B[0] = gather_s<ORDER>(g, f.Br, xa, ya - 0.5);
    B[1] = gather_s<ORDER>(g, f.Bth, xa - 0.5, ya);
    B[2] = gather_s<ORDER>(g, f.Bph, xa - 0.5, ya - 0.5);
  }

  // ---- Boris (full dt) at x^n, then geodesic predictor + K correctors (Eq.14, 15) ----
  const double r0 = exp(x1);
  double s0, c0;
  sincos(x2, &s0, &c0);
  const Pos p0 = make_pos(g, r0, s0, c0);
  const double alpha0 = p0.h * rsqrt_nr(p0.h);
  double ur = ptc.u1[k], ut = ptc.u2[k], up = ptc.u3[k];
  if (pusher == 1) vay(g, p0, alpha0, sgn, dt, D, B, ur, ut, up);
  else boris(g, p0, alpha0, sgn, dt, D, B, ur, ut, up);
  double Xr0, Xt0, Xp0, Ur0, Ut0;
  geodesic_rhs(g, p0, photon ? 0.0 : p0.zp1, ur, ut, up, Xr0, Xt0, Xp0, Ur0, Ut0);
  double dr = Xr0 * dt, dth = Xt0 * dt, dph = Xp0 * dt;
  double vr = fma(Ur0, dt, ur), vt = fma(Ut0, dt, ut);
  const double hdt = 0.5 * dt;
  for (int ci = 0; ci < K; ++ci) {
    double s, c;
    sincos(x2 + dth, &s, &c);
    const Pos p1 = make_pos(g, r0 + dr, s, c);
    double Xr, Xt, Xp, Ur, Ut;
    geodesic_rhs(g, p1, photon ? 0.0 : p1.zp1, vr, vt, up, Xr, Xt, Xp, Ur, Ut);
    dr = hdt * (Xr + Xr0);
    dth = hdt * (Xt + Xt0);
    dph = hdt * (Xp + Xp0);
    vr = fma(hdt, Ur + Ur0, ur);
    vt = fma(hdt, Ut + Ut0, ut);
  }
  const double x1n = log(r0 + dr), ph = ptc.x3[k] + dph;
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
  const double Q = sgn * ptc.w[k], vphi = Q * dph * idt;
  const double xb = (x1n - g.xi_in) * g.inv_dxi, yb = th_dep * g.inv_dth;
  const int ilo = (int)floor(fmin(xa, xb)) - EXT, ihi = (int)floor(fmax(xa, xb)) + 1 + EXT;
  const int jlo = (int)floor(fmin(ya, yb)) - EXT, jhi = (int)floor(fmax(ya, yb)) + 1 + EXT;
  if (ihi - ilo > 3 + 2 * EXT || jhi - jlo > 3 + 2 * EXT) { if (status) atomicOr(status, GRPIC_STATUS_FAR_MOVE); }
  if (ilo < -g.ng || ihi > g.nr + g.ng || jlo < -g.ng || jhi > g.nth + g.ng) {
    if (status) atomicOr(status, GRPIC_STATUS_OFFGRID);
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
  if (shape_order == 3)
    push_deposit_general_kernel<3><<<(unsigned)grid, 128, 0, st>>>(ctx->g, *ptc, *fields, *flux, dt,
                                                                   ctx->p.geo_iters, pusher, status);
  else
    push_deposit_general_kernel<1><<<(unsigned)grid, 128, 0, st>>>(ctx->g, *ptc, *fields, *flux, dt,
                                                                   ctx->p.geo_iters, pusher, status);
  grpic_count_launches(1);
  return grpic_launch_ok();
}

extern "C" int grpic_push_deposit_spline3(grpic_ctx* ctx, grpic_particles* ptc, const grpic_fields* fields,
                                          grpic_current* flux, double dt, uint32_t* status, void* stream) {
  return grpic_push_deposit_variant(ctx, ptc, fields, flux, dt, 3, 0, status, stream);
}
