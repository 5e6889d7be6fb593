// Flux post-processing: fold of theta ghost rows, binomial filter, division by the area
// elements, and the vertex charge density used by the continuity check.
#include <math.h>

#include "grpic_internal.cuh"

namespace {

// Fold the ghost rows onto their mirror rows (particles do not cross the axis):
// even parity for node-located F_r, F_ph, rho; odd for the half-staggered F_th.  One thread
// per padded column.
__global__ void fold_kernel(GridDev g, double* Fr, double* Fth, double* Fph) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x - g.ng;
  if (i > g.nr + g.ng) return;
  for (int gq = 1; gq <= g.ng; ++gq) {
    if (Fr) {
      Fr[g.idx(i, gq)] += Fr[g.idx(i, -gq)];
      Fr[g.idx(i, g.nth - gq)] += Fr[g.idx(i, g.nth + gq)];
      Fr[g.idx(i, -gq)] = 0.0;
      Fr[g.idx(i, g.nth + gq)] = 0.0;
    }
    if (Fph) {
      Fph[g.idx(i, gq)] += Fph[g.idx(i, -gq)];
      Fph[g.idx(i, g.nth - gq)] += Fph[g.idx(i, g.nth + gq)];
      Fph[g.idx(i, -gq)] = 0.0;
      Fph[g.idx(i, g.nth + gq)] = 0.0;
    }
    if (Fth) {
      Fth[g.idx(i, gq - 1)] -= Fth[g.idx(i, -gq)];
      Fth[g.idx(i, g.nth - gq)] -= Fth[g.idx(i, g.nth - 1 + gq)];
      Fth[g.idx(i, -gq)] = 0.0;
      Fth[g.idx(i, g.nth - 1 + gq)] = 0.0;
    }
  }
  if (Fth) Fth[g.idx(i, g.nth + g.ng)] = 0.0;
}

// One (1,2,1)x(1,2,1)/16 pass, src -> dst, for the three flux arrays (blockIdx.z).
__global__ void filter_kernel(GridDev g, const double* s0, const double* s1, const double* s2,
                              double* d0, double* d1, double* d2) {
  const int c = blockIdx.z;
  const double* S = c == 0 ? s0 : c == 1 ? s1 : s2;
  double* Dst = c == 0 ? d0 : c == 1 ? d1 : d2;
  const int ii = blockIdx.x * blockDim.x + threadIdx.x;
  const int jj = blockIdx.y;
  if (ii >= g.pitch) return;
  const int i = ii - g.i0, j = jj - g.j0;
  const bool half = (c == 1);
  const double par = half ? -1.0 : 1.0;
  const int jhi = half ? g.nth - 1 : g.nth;
  double out = 0.0;
  if (i >= -g.ng && i <= g.nr + g.ng && j >= 0 && j <= jhi) {
    const double wgt[3] = {1.0, 2.0, 1.0};
#pragma unroll
    for (int dj = -1; dj <= 1; ++dj) {
      int jn = j + dj;
      double sign = 1.0;
      if (!half) {
        if (jn < 0) { jn = -jn; sign = par; }
        if (jn > jhi) { jn = 2 * g.nth - jn; sign = par; }
      } else {
        if (jn < 0) { jn = -1 - jn; sign = par; }
        if (jn > jhi) { jn = 2 * g.nth - 1 - jn; sign = par; }
      }
      double row = 0.0;
#pragma unroll
      for (int di = -1; di <= 1; ++di) {
        const int in = min(max(i + di, -g.ng), g.nr + g.ng);
        row += wgt[di + 1] * __ldg(S + g.idx(in, jn));
      }
      out += sign * wgt[dj + 1] * row;
    }
    out *= (1.0 / 16.0);
  }
  Dst[(size_t)jj * g.pitch + ii] = out;
}

// J^r = F_r/A^D_r, J^th = F_th/A^D_th, J^ph = F_ph/(dphi A^D_ph)
__global__ void normalise_kernel(GridDev g, const double* s0, const double* s1, const double* s2,
                                 double* d0, double* d1, double* d2) {
  const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= g.size()) return;
  const double idphi = 1.0 / g.dphi;
  d0[k] = s0[k] * (__ldg(g.iADr + k) * idphi);
  d1[k] = s1[k] * (__ldg(g.iADth + k) * idphi);
  d2[k] = s2[k] * (__ldg(g.iADph + k) * idphi);
}

__global__ void rho_kernel(GridDev g, grpic_particles ptc, double* rho) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= ptc.n) return;
  const uint32_t flag = ptc.flag[k];
  if (flag & (2u | 4u)) return;   // removed, or photon (no charge)
  const double Q = ((flag & 1u) ? 1.0 : -1.0) * ptc.w[k];
  const double x = (ptc.x1[k] - g.xi_in) * g.inv_dxi, y = ptc.x2[k] * g.inv_dth;
  const double fi = floor(x), fj = floor(y);
  const int i = (int)fi, j = (int)fj;
  if (i < -g.ng || i + 1 > g.nr + g.ng || j < -g.ng || j + 1 > g.nth + g.ng) return;
  const double wx = x - fi, wy = y - fj;
  const size_t b = g.idx(i, j);
  atomicAdd(rho + b, Q * (1.0 - wx) * (1.0 - wy));
  atomicAdd(rho + b + 1, Q * wx * (1.0 - wy));
  atomicAdd(rho + b + g.pitch, Q * (1.0 - wx) * wy);
  atomicAdd(rho + b + g.pitch + 1, Q * wx * wy);
}

__global__ void rho_divide_kernel(GridDev g, double* rho) {
  const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= g.size()) return;
  rho[k] *= __ldg(g.iADph + k) / g.dphi;
}

}  // namespace

extern "C" {

int grpic_finalize_current(grpic_ctx* ctx, grpic_current* J, int32_t filter_passes, void* stream) {
  if (!ctx || !J || !J->Fr || !J->Fth || !J->Fph || filter_passes < 0) return GRPIC_ERR_ARG;
  const GridDev& g = ctx->g;
  const size_t n2 = g.size();
  cudaStream_t st = (cudaStream_t)stream;
  if (filter_passes > 0 && (!ctx->ws || ctx->ws_bytes < 3 * n2 * sizeof(double)))
    return GRPIC_ERR_WORKSPACE;
  fold_kernel<<<(g.nr + 1 + 2 * g.ng + 127) / 128, 128, 0, st>>>(g, J->Fr, J->Fth, J->Fph);
  double* a[3] = {J->Fr, J->Fth, J->Fph};
  double* b[3] = {(double*)ctx->ws, (double*)ctx->ws + n2, (double*)ctx->ws + 2 * n2};
  double** src = a;
  double** dst = b;
  for (int p = 0; p < filter_passes; ++p) {
    dim3 grid((g.pitch + 127) / 128, g.rows, 3);
    filter_kernel<<<grid, 128, 0, st>>>(g, src[0], src[1], src[2], dst[0], dst[1], dst[2]);
    double** t = src; src = dst; dst = t;
  }
  normalise_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>(g, src[0], src[1], src[2], J->Fr,
                                                                 J->Fth, J->Fph);
  grpic_count_launches(2 + filter_passes);
  return grpic_launch_ok();
}

int grpic_deposit_rho(grpic_ctx* ctx, const grpic_particles* ptc, double* rho, int32_t divide,
                      void* stream) {
  if (!ctx || !ptc || !rho || ptc->n < 0) return GRPIC_ERR_ARG;
  if (ptc->n > 0 && (!ptc->x1 || !ptc->x2 || !ptc->w || !ptc->flag)) return GRPIC_ERR_ARG;
  const GridDev& g = ctx->g;
  cudaStream_t st = (cudaStream_t)stream;
  GRPIC_CUDA_OK(cudaMemsetAsync(rho, 0, g.size() * sizeof(double), st));
  if (ptc->n > 0) {
    const int64_t grid = (ptc->n + 255) / 256;
    if (grid > 0x7FFFFFFFLL) return GRPIC_ERR_ARG;
    rho_kernel<<<(unsigned)grid, 256, 0, st>>>(g, *ptc, rho);
  }
  fold_kernel<<<(g.nr + 1 + 2 * g.ng + 127) / 128, 128, 0, st>>>(g, rho, nullptr, nullptr);
  if (divide) rho_divide_kernel<<<(unsigned)((g.size() + 255) / 256), 256, 0, st>>>(g, rho);
  grpic_count_launches((ptc->n > 0 ? 2 : 1) + (divide ? 1 : 0));
  return grpic_launch_ok();
}

}  // extern "C"
