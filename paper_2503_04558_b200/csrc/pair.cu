// Simplified pair production of the paper's Section 4 (Eq.26): leptons above
// the threshold FIDO Lorentz factor emit a photon of fixed FIDO energy along their motion;
// photons convert into an e-/e+ pair with probability 1 - exp(-tau dt) per step.  New particles
// are appended in the order of their parents (warp ballot + device-wide scan), random numbers
// come from a counter-based Philox4x32-10 keyed by (seed; particle index, step), so the result
// does not depend on the launch shape.  Readings P1-P4: DESIGN.md.
#include <math.h>

#include "grpic_internal.cuh"

namespace {

// Philox4x32-10 (Salmon et al., SC'11): ten rounds of two 32x32->64 multiplies and key bumps.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t& o0, uint32_t& o1) {
#pragma unroll
  for (int round = 0; round < 10; ++round) {
    const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
    const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
    c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  o0 = c0; o1 = c1;
}
__device__ __forceinline__ double uniform53(uint64_t seed, uint32_t step, uint64_t index) {
  uint32_t o0, o1;
  philox4x32_10((uint32_t)index, (uint32_t)(index >> 32), step, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), o0,
                o1);
  const uint64_t bits = (((uint64_t)o0 << 32) | o1) >> 11;
  return (double)bits * (1.0 / 9007199254740992.0);
}

// gamma^ij u_i u_j at (r = exp(x1), theta)   (Appendix A)
__device__ __forceinline__ double fido_norm(const GridDev& g, double x1, double x2, double ur, double ut,
                                            double up) {
  const double r = exp(x1);
  double s, c;
  sincos(x2, &s, &c);
  const double rho2 = fma(g.a2 * c, c, r * r);
  const double R = 1.0 / rho2;
  const double beta = g.twoM * r / (rho2 + g.twoM * r);
  const double gu_rr = (r * r + g.a2) * R - beta, gu_pp = R / (s * s), gu_rp = g.a * R;
  return gu_rr * ur * ur + R * ut * ut + gu_pp * up * up + 2.0 * gu_rp * ur * up;
}

struct Event {           // what one particle does in this pass
  double child_scale;    // 0: nothing
  double parent_scale;
  uint32_t child_flag, parent_flag;
};
__device__ __forceinline__ Event decide(const GridDev& g, const grpic_particles& P, int64_t k,
                                        const grpic_pair_params& pp) {
  Event e = {0.0, 1.0, 0u, 0u};
  const uint32_t flag = P.flag[k];
  e.parent_flag = flag;
  if (flag & 2u) return e;
  const double N = fido_norm(g, P.x1[k], P.x2[k], P.u1[k], P.u2[k], P.u3[k]);
  if (!(flag & 4u)) {                                  // lepton: emission at the threshold
    const double Gamma = sqrt(1.0 + N), umag = sqrt(N);
    if (Gamma >= pp.gamma_thr && umag > pp.eps_ph) {
      e.child_scale = pp.eps_ph / umag;
      e.parent_scale = 1.0 - pp.eps_ph / umag;
      e.child_flag = 4u;
    }
  } else {                                             // photon: conversion, Eq.(26)
    const double E = sqrt(N), Gl = 0.5 * E;
    if (uniform53(pp.seed, pp.step, (uint64_t)k) < pp.p_convert && Gl > 1.0) {
      e.child_scale = e.parent_scale = sqrt(Gl * Gl - 1.0) / E;
      e.parent_flag = 0u;
      e.child_flag = 1u;
    }
  }
  return e;
}

// pass 1: number of children per 32-particle tile, and which lanes have one (the second pass reads the
// particle data of those lanes only: 44 B per particle once instead of twice; 2.53 -> see
// profiles/r02_late_experiments.md)
__global__ void __launch_bounds__(256)
pair_count_kernel(const __grid_constant__ GridDev g, const __grid_constant__ grpic_particles P,
                  const __grid_constant__ grpic_pair_params pp, uint32_t* counts, uint32_t* masks) {
  const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
  bool child = false;
  if (k < P.n) child = decide(g, P, k, pp).child_scale != 0.0;
  const uint32_t b = __ballot_sync(0xffffffffu, child);
  if ((threadIdx.x & 31) == 0 && k < P.n) { counts[k >> 5] = __popc(b); masks[k >> 5] = b; }
}
// pass 2: children to n + offsets[tile] + rank, parents updated in place
__global__ void __launch_bounds__(256)
pair_apply_kernel(const __grid_constant__ GridDev g, const __grid_constant__ grpic_particles P,
                  const __grid_constant__ grpic_pair_params pp, const uint32_t* offsets,
                  const uint32_t* __restrict__ masks, uint32_t ntiles, int64_t capacity, int64_t* n_new,
                  uint32_t* status) {
  const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
  const int lane = threadIdx.x & 31;
  const int64_t tile = k >> 5;
  if (k >= P.n) return;
  const uint32_t b = masks[tile];                      // the first pass's decisions (same arithmetic below)
  const bool child = (b >> lane) & 1u;
  if (k < P.n && tile == (int64_t)ntiles - 1 && lane == 0) {
    const int64_t total = P.n + (int64_t)offsets[tile] + __popc(b);
    *n_new = total < capacity ? total : capacity;
    if (total > capacity && status) atomicOr(status, GRPIC_STATUS_CAPACITY);
  }
  if (!child) return;
  const Event e = decide(g, P, k, pp);
  const double ur = P.u1[k], ut = P.u2[k], up = P.u3[k];
  const int64_t d = P.n + (int64_t)offsets[tile] + __popc(b & ((1u << lane) - 1u));
  if (d >= capacity) return;      // P5: an event whose child has no room does not happen (parent unchanged)
  P.x1[d] = P.x1[k]; P.x2[d] = P.x2[k]; P.x3[d] = P.x3[k];
  P.u1[d] = ur * e.child_scale; P.u2[d] = ut * e.child_scale; P.u3[d] = up * e.child_scale;
  P.w[d] = P.w[k]; P.cell[d] = P.cell[k]; P.flag[d] = e.child_flag;
  P.u1[k] = ur * e.parent_scale; P.u2[k] = ut * e.parent_scale; P.u3[k] = up * e.parent_scale;
  P.flag[k] = e.parent_flag;
}

}  // namespace

extern "C" int grpic_pair_production(grpic_ctx* ctx, grpic_particles* ptc, int64_t capacity,
                                     const grpic_pair_params* params, int64_t* n_new, uint32_t* status,
                                     void* stream) {
  if (!ctx || !ptc || !params || !n_new || ptc->n < 0 || capacity < ptc->n) return GRPIC_ERR_ARG;
  if (!(params->p_convert >= 0.0 && params->p_convert <= 1.0) || !(params->eps_ph > 0.0)) return GRPIC_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = ptc->n;
  if (n == 0) {
    GRPIC_CUDA_OK(cudaMemsetAsync(n_new, 0, sizeof(int64_t), st));
    return GRPIC_OK;
  }
  if (!ptc->x1 || !ptc->x2 || !ptc->x3 || !ptc->u1 || !ptc->u2 || !ptc->u3 || !ptc->w || !ptc->cell ||
      !ptc->flag || capacity > 0xFFFFFFF0LL)
    return GRPIC_ERR_ARG;
  const size_t ntiles = (size_t)((n + 31) / 32);
  const size_t need = (2 * ntiles + ntiles / 2048 + 4096) * sizeof(uint32_t);
  if (!ctx->ws || ctx->ws_bytes < need) return GRPIC_ERR_WORKSPACE;
  uint32_t* offsets = (uint32_t*)ctx->ws;
  uint32_t* masks = offsets + ntiles + ntiles / 2048 + 4096;
  const unsigned grid = (unsigned)((n + 255) / 256);
  pair_count_kernel<<<grid, 256, 0, st>>>(ctx->g, *ptc, *params, offsets, masks);
  int rc = grpic_exclusive_scan(offsets, ntiles, offsets + ntiles, st);
  if (rc != GRPIC_OK) return rc;
  pair_apply_kernel<<<grid, 256, 0, st>>>(ctx->g, *ptc, *params, offsets, masks, (uint32_t)ntiles, capacity, n_new,
                                          status);
  grpic_count_launches(2);
  return grpic_launch_ok();
}
