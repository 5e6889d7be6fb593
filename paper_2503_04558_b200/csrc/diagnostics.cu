// Per-particle diagnostics in Boyer-Lindquist coordinates and in the FIDO frame (PAPER.md:458-474,
// Appendix A (A6)-(A7)).  The Kerr-Schild state (ln r, theta, phi, u_r, u_theta,
// u_phi) of every live particle is turned into
//   E_inf  = -u_t = alpha^2 u^0 - beta^r u_r            (energy at infinity, conserved on geodesics),
//   Gamma  = alpha u^0                                  (Lorentz factor seen by the FIDO),
//   u_r^BL = u_r^KS - (2 M r E_inf - a u_phi) / Delta   ((A6): dt_KS = dt_BL + 2Mr/Delta dr, dphi_KS =
//                                                        dphi_BL + a/Delta dr; u_t, u_theta, u_phi unchanged),
//   phi_BL = phi_KS - a / (2 sqrt(M^2 - a^2)) ln|(r - r_+) / (r - r_-)|          ((A7)).
// One thread per particle; removed particles get NaN.  Parity-level kernel (HBM-bound, 52 B in, 32 B out).
#include <math.h>

#include "grpic_internal.cuh"

namespace {

__global__ void __launch_bounds__(256)
ks_to_bl_kernel(const __grid_constant__ GridDev g, const __grid_constant__ grpic_particles P, double* E_inf,
                double* gamma_fido, double* ur_bl, double* phi_bl) {
  const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (k >= P.n) return;
  const uint32_t flag = P.flag[k];
  double E = nan(""), Gam = E, urb = E, phb = E;
  if (!(flag & 2u)) {
    const double r = exp(P.x1[k]);
    double s, c;
    sincos(P.x2[k], &s, &c);
    const double ur = P.u1[k], ut = P.u2[k], up = P.u3[k];
    const double rho2 = fma(g.a2 * c, c, r * r), z = g.twoM * r / rho2;
    const double alpha2 = 1.0 / (1.0 + z), beta = z * alpha2;
    // gamma^ij u_i u_j  (A4)
    const double N = ((r * r + g.a2) / rho2 - beta) * ur * ur + ut * ut / rho2 + up * up / (rho2 * s * s) +
                     2.0 * g.a / rho2 * ur * up;
    const double eps = (flag & 4u) ? 0.0 : 1.0;
    const double u0 = sqrt((eps + N) / alpha2);
    E = alpha2 * u0 - beta * ur;
    Gam = sqrt(alpha2) * u0;
    const double Delta = r * r - g.twoM * r + g.a2;
    urb = ur - (g.twoM * r * E - g.a * up) / Delta;
    const double M = 0.5 * g.twoM, root = sqrt(M * M - g.a2);
    phb = P.x3[k] - (root > 0.0 ? g.a / (2.0 * root) * log(fabs((r - (M + root)) / (r - (M - root)))) : 0.0);
  }
  if (E_inf) E_inf[k] = E;
  if (gamma_fido) gamma_fido[k] = Gam;
  if (ur_bl) ur_bl[k] = urb;
  if (phi_bl) phi_bl[k] = phb;
}

}  // namespace

extern "C" int grpic_ks_to_bl(grpic_ctx* ctx, const grpic_particles* ptc, double* E_inf, double* gamma_fido,
                              double* ur_bl, double* phi_bl, void* stream) {
  if (!ctx || !ptc || ptc->n < 0) return GRPIC_ERR_ARG;
  if (ptc->n == 0) return GRPIC_OK;
  if (!ptc->x1 || !ptc->x2 || !ptc->x3 || !ptc->u1 || !ptc->u2 || !ptc->u3 || !ptc->flag) return GRPIC_ERR_ARG;
  ks_to_bl_kernel<<<(unsigned)((ptc->n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(ctx->g, *ptc, E_inf, gamma_fido,
                                                                                     ur_bl, phi_bl);
  grpic_count_launches(1);
  return grpic_launch_ok();
}
