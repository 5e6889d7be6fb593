// Fused GR particle push + charge-conserving current deposit (sm_100a).
//
// One thread per particle.  All Kerr-Schild metric terms (lapse, shift, spatial metric, inverse
// metric and the r/theta derivatives entering Eq.12) are computed inline in registers from
// (r, sin theta, cos theta) with ONE reciprocal per evaluation point; position-only terms are
// shared between the Boris rotation and the first geodesic right-hand side.  The corrector
// iterates get sin/cos by angle addition from the start point and the new ln r by a short
// atanh series, so a particle-step costs one exp, one sincos and no log on the common path.
// Closed forms: Appendix A with M restored; derivative forms are this
// file's own.
//
// Deposit (Eq.21-23): every particle adds the fluxes of its move to the
// 3x3-node window anchored at the lower of its old and new cell (2x3 F_r faces, 3x2 F_theta
// faces, 3x3 F_phi nodes) with RED.E.ADD.F64; the slots that vanish unless the move crosses a
// cell face are grouped behind two tests, so a particle issues 8 / 13 / 21 REDs and no
// per-slot branch.  Measured on B200 (profiles/r01c): the cell sort decays within a few steps
// (particles move up to half a cell per step), so schemes that reduce runs of equal cell inside
// a warp before the atomics (v2/v3 of this file) only pay right after a sort, while their
// per-slot zero tests cost ~200 control instructions per particle afterwards.
#include <math.h>
#include <stdlib.h>

#include "grpic_internal.cuh"
#include "push_math.cuh"

namespace {

// CTA size and the two occupancy settings (resident CTAs per SM) the launcher chooses between.
// Measured at 1e8 particles, compacting / in place (ms): 256 threads x 2: 6.87 / 6.53; 128 x 4: 6.70 / 6.36,
// 128 x 5: 7.11 / 6.22; 64 x 8: 6.62 / 6.27, 64 x 10: 6.99 / 6.11; 32 x 16: 7.00 / 6.56.
#ifndef GRPIC_PD_BLOCK
#define GRPIC_PD_BLOCK 64
#endif
#ifndef GRPIC_PD_MA
#define GRPIC_PD_MA 8      // 126 registers per thread: the compacting variant
#endif
#ifndef GRPIC_PD_MB
#define GRPIC_PD_MB 10     // 96 registers per thread: the in-place variant
#endif
constexpr int kBlock = GRPIC_PD_BLOCK;

// Charge-conserving deposit of one move (Eq.21-23) on the 3x3-node window anchored at the
// lower of the old and new cell in each direction: a move of less than one cell touches at
// most two cells per direction, so 2 F_r faces x 3 rows, 3 columns x 2 F_theta faces and 3x3
// F_phi nodes hold every non-zero flux.  Inputs per direction: the in-cell fractions of the old
// and new position (fa, fb in [0,1)) and which of the window's two cells each lies in (oa, ob in
// {0,1}).  The CIC shapes on the three nodes are then (1-f, f, 0) or (0, 1-f, f): plain selects,
// no max() (a double fmax costs six instructions for its NaN rules).  No per-slot zero test (each
// costs a divergent branch around the atomic); issuing all 21 REDs unconditionally is LSU-bound
// (12.5 ms vs 7.1 ms at 1e8), so the slots that vanish unless a cell face is crossed are grouped.
__device__ __forceinline__ void deposit_local(const grpic_current& J, uint32_t anchor, uint32_t pitch,
                                              double Q, double vphi, double idt, double fxa, double fya,
                                              double fxb, double fyb, bool oax, bool oay, bool obx,
                                              bool oby) {
  const double gxa = 1.0 - fxa, gya = 1.0 - fya, gxb = 1.0 - fxb, gyb = 1.0 - fyb;
  const double Sa0 = oax ? 0.0 : gxa, Sa1 = oax ? gxa : fxa, Sa2 = oax ? fxa : 0.0;
  const double Sb0 = obx ? 0.0 : gxb, Sb1 = obx ? gxb : fxb, Sb2 = obx ? fxb : 0.0;
  const double Ta0 = oay ? 0.0 : gya, Ta1 = oay ? gya : fya, Ta2 = oay ? fya : 0.0;
  const double Tb0 = oby ? 0.0 : gyb, Tb1 = oby ? gyb : fyb, Tb2 = oby ? fyb : 0.0;
  const bool cx = oax != obx, cy = oay != oby;
  const double hq = -0.5 * Q * idt;
  // prefix sums of the shape differences over the two faces (Eq.21); the third vanishes
  const double Px0 = Sb0 - Sa0, Px1 = Sa2 - Sb2;
  const double Py0 = Tb0 - Ta0, Py1 = Ta2 - Tb2;
  const double Ay0 = hq * (Tb0 + Ta0), Ay1 = hq * (Tb1 + Ta1), Ay2 = hq * (Tb2 + Ta2);
  const double Ax0 = hq * (Sb0 + Sa0), Ax1 = hq * (Sb1 + Sa1), Ax2 = hq * (Sb2 + Sa2);
  // F_phi (Eq.23) = Sb_i U_j + Sa_i V_j
  const double c3 = vphi * (1.0 / 3.0), c6 = vphi * (1.0 / 6.0);
  const double U0 = fma(c3, Tb0, c6 * Ta0), U1 = fma(c3, Tb1, c6 * Ta1), U2 = fma(c3, Tb2, c6 * Ta2);
  const double V0 = fma(c3, Ta0, c6 * Tb0), V1 = fma(c3, Ta1, c6 * Tb1), V2 = fma(c3, Ta2, c6 * Tb2);
  double* fr = J.Fr + anchor;
  double* ft = J.Fth + anchor;
  double* fp = J.Fph + anchor;
  const uint32_t p2 = 2u * pitch;
  {
    // slots that vanish unless the move crosses a cell face in xi (cx) / theta (cy) are
    // grouped behind those two tests: 8 always, +5 if cx, +5 if cy, +3 if both
    atomicAdd(fr, Ay0 * Px0);          atomicAdd(fr + pitch, Ay1 * Px0);
    atomicAdd(ft, Ax0 * Py0);          atomicAdd(ft + 1, Ax1 * Py0);
    atomicAdd(fp, fma(Sb0, U0, Sa0 * V0));          atomicAdd(fp + 1, fma(Sb1, U0, Sa1 * V0));
    atomicAdd(fp + pitch, fma(Sb0, U1, Sa0 * V1));  atomicAdd(fp + pitch + 1, fma(Sb1, U1, Sa1 * V1));
    if (cx) {
      atomicAdd(fr + 1, Ay0 * Px1);    atomicAdd(fr + pitch + 1, Ay1 * Px1);
      atomicAdd(ft + 2, Ax2 * Py0);
      atomicAdd(fp + 2, fma(Sb2, U0, Sa2 * V0));    atomicAdd(fp + pitch + 2, fma(Sb2, U1, Sa2 * V1));
    }
    if (cy) {
      atomicAdd(fr + p2, Ay2 * Px0);
      atomicAdd(ft + pitch, Ax0 * Py1);  atomicAdd(ft + pitch + 1, Ax1 * Py1);
      atomicAdd(fp + p2, fma(Sb0, U2, Sa0 * V2));   atomicAdd(fp + p2 + 1, fma(Sb1, U2, Sa1 * V2));
      if (cx) {
        atomicAdd(fr + p2 + 1, Ay2 * Px1);
        atomicAdd(ft + pitch + 2, Ax2 * Py1);
        atomicAdd(fp + p2 + 2, fma(Sb2, U2, Sa2 * V2));
      }
    }
  }
}

// ---- TMA (cp.async.bulk) + mbarrier plumbing for the double-buffered particle tiles ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    if (!ok) __nanosleep(64);                       // do not burn issue slots other warps can use
  } while (!ok);
}
// The particle stream (12.8 GB per step at 1e8) is read and written once: it is marked
// evict-first in L2 so that the field and flux lines the gather and the REDs revisit stay resident.
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}

// One warp tile of particle input staged in shared memory (structure of arrays, 32 particles).
constexpr int kWarps = kBlock / 32;
#ifndef GRPIC_PD_STAGES
#define GRPIC_PD_STAGES 3
#endif
constexpr int kPdStages = GRPIC_PD_STAGES;   // particle tiles in flight per CTA
struct __align__(128) PtcTile {
  double x1[kBlock], x2[kBlock], x3[kBlock], u1[kBlock], u2[kBlock], u3[kBlock], w[kBlock];
  uint32_t flag[kBlock];
  uint32_t dest[kBlock];   // COMPACT: output index of each particle (written by its own thread, not by TMA)
};
constexpr uint32_t kTileBytes = 7u * kBlock * 8u + kBlock * 4u;

// Persistent kernel.  A CTA walks the kBlock-particle tiles blockIdx.x, + gridDim.x, ...; a ring of
// shared-memory stages holds the particle state of the current and the next tiles, each filled by
// eight 1-D bulk TMA copies (block-uniform addresses: no per-warp address arithmetic).  There is
// no block-wide barrier in the loop: the warps run independently, each waits on the
// stage's mbarrier for its data, counts itself out of the stage when it has read it, and the
// last warp out refills the stage with the tile kPdStages steps ahead.  A warp that takes a slow path
// (far deposit, large-angle sincos) delays the others by at most one tile.  The last, partial
// tile (n % kBlock != 0) is staged with plain loads.
//
// COMPACT: the results are stored to `dst` at offsets[tile] + rank among the tile's live lanes
// (offsets = exclusive scan of the per-tile live counts of `ptc`), i.e. particles already
// flagged removed are squeezed out on the way, order preserved; the weight travels along.
// Otherwise dst == ptc and the update is in place.
template <int MINB, bool COMPACT, int KT>
__global__ void __launch_bounds__(kBlock, MINB)
push_deposit_kernel(const __grid_constant__ GridDev g, const __grid_constant__ grpic_particles ptc,
                    const __grid_constant__ grpic_particles dst, const uint32_t* __restrict__ offsets,
                    int64_t* n_alive, const __grid_constant__ grpic_fields f,
                    const __grid_constant__ grpic_current J, double dt, int K, uint32_t* status) {
  __shared__ PtcTile tiles[kPdStages];
  __shared__ __align__(8) uint64_t full[kPdStages];
  __shared__ uint32_t done[kPdStages];                       // warps that have finished reading a stage
  // read once (volatile: the compiler otherwise re-reads SR_TID.X, ~20 cycles each, when short of registers)
  uint32_t tid_x;
  asm volatile("mov.u32 %0, %%tid.x;" : "=r"(tid_x));
  const int tid = tid_x, lane = tid_x & 31, warp = tid_x >> 5;
  // all particle indices fit 32 bits (the C entry rejects n > 0xFFFFFFF0): one-instruction addressing
  const uint32_t n32 = (uint32_t)ptc.n;
  const uint32_t ntiles = (n32 + kBlock - 1) / kBlock;
  const uint32_t ntiles32 = (n32 + 31) / 32;           // COMPACT: offsets are per 32-particle tile
  const uint32_t tstride = gridDim.x;
  const double idt = 1.0 / dt;

  const uint64_t stream_policy = l2_evict_first_policy();
  auto issue = [&](uint32_t tile, int stage) {      // one thread; full tiles only
    const uint32_t k0 = tile * kBlock;
    if (tile >= ntiles || k0 + kBlock > n32) return;
    PtcTile& T = tiles[stage];
    uint64_t* bar = &full[stage];
    mbar_expect_tx(bar, kTileBytes);
    tma_load_1d(T.x1, ptc.x1 + k0, kBlock * 8, bar, stream_policy);
    tma_load_1d(T.x2, ptc.x2 + k0, kBlock * 8, bar, stream_policy);
    tma_load_1d(T.x3, ptc.x3 + k0, kBlock * 8, bar, stream_policy);
    tma_load_1d(T.u1, ptc.u1 + k0, kBlock * 8, bar, stream_policy);
    tma_load_1d(T.u2, ptc.u2 + k0, kBlock * 8, bar, stream_policy);
    tma_load_1d(T.u3, ptc.u3 + k0, kBlock * 8, bar, stream_policy);
    tma_load_1d(T.w, ptc.w + k0, kBlock * 8, bar, stream_policy);
    tma_load_1d(T.flag, ptc.flag + k0, kBlock * 4, bar, stream_policy);
  };
  const uint32_t tile0 = blockIdx.x;
  if (tid == 0) {
#pragma unroll
    for (int q = 0; q < kPdStages; ++q) { mbar_init(&full[q], 1); done[q] = 0; }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
#pragma unroll
    for (int q = 0; q < kPdStages; ++q) issue(tile0 + q * tstride, q);
  }
  __syncthreads();                                  // the only block barrier: before the loop

  int it = 0;
  // COMPACT: output offset of this warp's 32-particle tile, loaded one tile ahead
  uint32_t obase_next = (COMPACT && tile0 * kWarps + warp < ntiles32) ? offsets[tile0 * kWarps + warp] : 0u;
  for (uint32_t tile = tile0; tile < ntiles; tile += tstride, ++it) {
  const int stage = it % kPdStages;
  PtcTile& T = tiles[stage];
  const uint32_t k = tile * kBlock + tid;
  const uint32_t tile32 = tile * kWarps + warp;     // this warp's 32-particle tile
  if (tile * kBlock + kBlock <= n32) {
    mbar_wait(&full[stage], (uint32_t)(it / kPdStages) & 1u);
  } else {                                          // partial last tile: every thread stages its own slot
    if (k < n32) {
      T.x1[tid] = ptc.x1[k]; T.x2[tid] = ptc.x2[k]; T.x3[tid] = ptc.x3[k];
      T.u1[tid] = ptc.u1[k]; T.u2[tid] = ptc.u2[k]; T.u3[tid] = ptc.u3[k];
      T.w[tid] = ptc.w[k];
      T.flag[tid] = ptc.flag[k];
    } else {
      T.flag[tid] = 2u;
    }
    __syncwarp();
  }
  const uint32_t flag = T.flag[tid];
  const bool active = !(flag & 2u);
  if (COMPACT) {
    // where this particle's result goes: offsets[tile32] + rank among the live lanes, parked in
    // the tile's shared memory instead of a register that would live across the whole push
    const uint32_t live = __ballot_sync(0xffffffffu, active);
    const uint32_t obase = obase_next;
    if (tile32 + tstride * kWarps < ntiles32) obase_next = offsets[tile32 + tstride * kWarps];
    if (tile32 == ntiles32 - 1 && lane == 0) *n_alive = (int64_t)obase + __popc(live);
    T.dest[tid] = obase + __popc(live & ((1u << lane) - 1u));
  }

  if (active) {
    const double x1 = T.x1[tid], x2 = T.x2[tid];
    // species: charge sign of e-/e+; a photon (bit2) feels no Lorentz force
    // (sgn = 0 makes the Boris step the exact identity), has eps = 0 and carries no charge
    const bool photon = (flag & 4u) != 0;
    const double sgn = photon ? 0.0 : ((flag & 1u) ? 1.0 : -1.0);

    // ---- gather (first order, each component from its own staggered lattice): the 24
    // loads are issued first, exp / sincos / metric run while they are in flight ----
    const double xa = (x1 - g.xi_in) * g.inv_dxi, ya = x2 * g.inv_dth;
    const double fin = floor(xa), fjn = floor(ya);
    const int ia = (int)fin, ja = (int)fjn;
    const double fih = floor(xa - 0.5), fjh = floor(ya - 0.5);
    const int ih = (int)fih, jh = (int)fjh;
    const uint32_t bnn = (uint32_t)g.idx(ia, ja), bhn = (uint32_t)g.idx(ih, ja);
    const uint32_t bnh = (uint32_t)g.idx(ia, jh), bhh = (uint32_t)g.idx(ih, jh);
    double G[6][4];
    {
      const double* F6[6] = {f.Dr, f.Dth, f.Dph, f.Br, f.Bth, f.Bph};
      const uint32_t b6[6] = {bhn, bnh, bnn, bnh, bhn, bhh};
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        G[c][0] = __ldg(F6[c] + b6[c]);
        G[c][1] = __ldg(F6[c] + b6[c] + 1);
        G[c][2] = __ldg(F6[c] + b6[c] + g.pitch);
        G[c][3] = __ldg(F6[c] + b6[c] + g.pitch + 1);
      }
    }

    // ---- metric at x^n ----
    const double r0 = exp(x1);
    double s0, c0;
    sincos(x2, &s0, &c0);
    const Pos p0 = make_pos(g, r0, s0, c0);
    const double alpha0 = p0.h * rsqrt_nr(p0.h);      // lapse at x^n

    double D[3], B[3];
    {
      double wxn = xa - fin;
      // scheduling fence: the interpolation (first use of the 24 loads above) may not start
      // before the position-only metric terms exist, so exp, sincos, the reciprocal and the
      // rsqrt of the lapse all run in the shadow of the gather's L2 latency
      asm volatile("" : "+d"(wxn) : "d"(p0.R), "d"(alpha0));
      const double wyn = ya - fjn, wxh = xa - 0.5 - fih, wyh = ya - 0.5 - fjh;
      const double wx6[6] = {wxh, wxn, wxn, wxn, wxh, wxh};
      const double wy6[6] = {wyn, wyh, wyn, wyh, wyn, wyh};
      double V6[6];
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        const double lo = fma(wx6[c], G[c][1] - G[c][0], G[c][0]);
        const double hi = fma(wx6[c], G[c][3] - G[c][2], G[c][2]);
        V6[c] = fma(wy6[c], hi - lo, lo);
      }
      D[0] = V6[0]; D[1] = V6[1]; D[2] = V6[2]; B[0] = V6[3]; B[1] = V6[4]; B[2] = V6[5];
    }

    // ---- Boris (full dt) at x^n ----
    double ur = T.u1[tid], ut = T.u2[tid], up = T.u3[tid];
    boris(g, p0, alpha0, sgn, dt, D, B, ur, ut, up);

    // ---- geodesic predictor + K correctors (Eq.14, 15) ----
    double Xr0, Xt0, Xp0, Ur0, Ut0;
    geodesic_rhs(g, p0, photon ? 0.0 : p0.zp1, ur, ut, up, Xr0, Xt0, Xp0, Ur0, Ut0);
    double dr = Xr0 * dt, dth = Xt0 * dt, dph = Xp0 * dt;      // increments from x^n
    double vr = fma(Ur0, dt, ur), vt = fma(Ut0, dt, ut);
    const double hdt = 0.5 * dt;
    const int KK = KT > 0 ? KT : K;                 // KT: compile-time corrector count (unrolled)
#pragma unroll
    for (int ci = 0; ci < KK; ++ci) {
      double s, c;
      if (fabs(dth) <= 0.001953125) sincos_shift<true>(s0, c0, dth, s, c);
      else if (fabs(dth) <= 0.06) sincos_shift<false>(s0, c0, dth, s, c);
      else sincos(x2 + dth, &s, &c);
      const Pos p1 = make_pos(g, r0 + dr, s, c);
      double Xr, Xt, Xp, Ur, Ut;
      geodesic_rhs(g, p1, photon ? 0.0 : p1.zp1, vr, vt, up, Xr, Xt, Xp, Ur, Ut);
      dr = hdt * (Xr + Xr0);
      dth = hdt * (Xt + Xt0);
      dph = hdt * (Xp + Xp0);
      vr = fma(hdt, Ur + Ur0, ur);
      vt = fma(hdt, Ut + Ut0, ut);
    }
    const double r = r0 + dr, ph = T.x3[tid] + dph;
    double th = x2 + dth;

    // ---- new logical position: ln r = x1 + 2 atanh(dr / (2 r0 + dr)) ----
    double x1n;
    {
      const double wq = dr * rcp_nr(r0 + r);
      if (fabs(wq) <= 0.03) {
        const double w2 = wq * wq;
        double pl = fma(w2, 1.0 / 11.0, 1.0 / 9.0);
        pl = fma(pl, w2, 1.0 / 7.0);
        pl = fma(pl, w2, 1.0 / 5.0);
        pl = fma(pl, w2, 1.0 / 3.0);
        const double at = fma(pl * w2, wq, wq);
        x1n = fma(2.0, at, x1);
      } else {
        x1n = log(r);
      }
    }
    // ---- reflection, removal, new cell ----
    const double th_dep = th;
    if (th < 0.0) { th = -th; vt = -vt; }
    if (th > M_PI) { th = 2.0 * M_PI - th; vt = -vt; }
    // new logical position (un-reflected), its cell and in-cell fractions
    const double xb = (x1n - g.xi_in) * g.inv_dxi, yb = th_dep * g.inv_dth;
    const double fib = floor(xb), fjb = floor(yb);
    const int ib = (int)fib, jb = (int)fjb;
    const double fxb = xb - fib, fyb = yb - fjb;
    uint32_t nflag = flag, ncell;
    const bool finite = isfinite(x1n) && isfinite(th) && isfinite(ph) && isfinite(vr) && isfinite(vt);
    const bool out = !finite || (x1n < g.xi_in) || (x1n >= g.xi_out);
    if (out) {
      nflag |= 2u;
      ncell = 0xFFFFFFFFu;
      if (!finite && status) atomicOr(status, GRPIC_STATUS_NONFINITE);
    } else {
      // cell = floor of the quotient; the product form decides unless it is within 1e-7 of
      // a cell edge, where the quotient itself is taken (same decision as a division)
      int ic = ib, jc = jb;
      if (fabs(fxb - 0.5) > 0.5 - 1e-7) ic = (int)floor((x1n - g.xi_in) / g.dxi);
      if (th != th_dep) {                             // reflected at an axis: recompute in theta
        const double cy = th * g.inv_dth, fc = floor(cy);
        jc = (int)fc;
        if (fabs(cy - fc - 0.5) > 0.5 - 1e-7) jc = (int)floor(th / g.dth);
      } else if (fabs(fyb - 0.5) > 0.5 - 1e-7) {
        jc = (int)floor(th / g.dth);
      }
      ic = min(max(ic, 0), g.nr - 1);
      jc = min(max(jc, 0), g.nth - 1);
      ncell = (uint32_t)(jc * g.nr + ic);
    }
    const uint32_t kd = COMPACT ? T.dest[tid] : k;
    __stcs(dst.x1 + kd, x1n); __stcs(dst.x2 + kd, th); __stcs(dst.x3 + kd, ph);   // streaming stores
    __stcs(dst.u1 + kd, vr); __stcs(dst.u2 + kd, vt); __stcs(dst.u3 + kd, up);
    if (COMPACT) __stcs(dst.w + kd, T.w[tid]);
    __stcs(dst.cell + kd, ncell);
    __stcs(dst.flag + kd, nflag);

    // ---- deposit: 3x3 window anchored at the lower of the old / new cell ----
    if (finite && !photon) {
      const double q = sgn * T.w[tid];
      const double vph = q * dph * idt;
      const int di = ib - ia, dj = jb - ja;
      if (di >= -1 && di <= 1 && dj >= -1 && dj <= 1) {
        const int iw = min(ia, ib), jw = min(ja, jb);
        deposit_local(J, (uint32_t)g.idx(iw, jw), (uint32_t)g.pitch, q, vph, idt, xa - fin, ya - fjn, fxb,
                      fyb, ia != iw, ja != jw, ib != iw, jb != jw);
      } else {
        deposit_far(&g, q, idt, vph, xa, xb, ya, yb, J.Fr, J.Fth, J.Fph, status);
      }
    }
  }
  // this warp is done with the stage; the last warp out refills it with the tile two steps ahead
  __syncwarp();
  if (lane == 0) {
    if (atomicAdd(&done[stage], 1u) == kWarps - 1) {
      atomicExch(&done[stage], 0u);
      issue(tile + kPdStages * tstride, stage);
    }
  }
  }
}

template <int MINB, bool COMPACT, int KT>
int launch_push_deposit(const grpic_ctx* ctx, const grpic_particles& ptc, const grpic_particles& dst,
                        const uint32_t* offsets, int64_t* n_alive, const grpic_fields& f,
                        const grpic_current& J, double dt, uint32_t* status, cudaStream_t st) {
  static int per_sm = 0;   // resident CTAs per SM of this instantiation
  if (per_sm == 0) {
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, push_deposit_kernel<MINB, COMPACT, KT>,
                                                      kBlock, 0) != cudaSuccess || per_sm < 1)
      per_sm = 1;
  }
  const int64_t nblocks = (ptc.n + kBlock - 1) / kBlock;
  const int64_t resident = (int64_t)ctx->sm_count * per_sm;
  const unsigned grid = (unsigned)(nblocks < resident ? nblocks : resident);
  push_deposit_kernel<MINB, COMPACT, KT><<<grid, kBlock, 0, st>>>(ctx->g, ptc, dst, offsets, n_alive, f, J,
                                                                  dt, ctx->p.geo_iters, status);
  return grpic_launch_ok();
}

template <bool COMPACT>
int dispatch_push_deposit(const grpic_ctx* ctx, const grpic_particles& ptc, const grpic_particles& dst,
                          const uint32_t* offsets, int64_t* n_alive, const grpic_fields& f,
                          const grpic_current& J, double dt, uint32_t* status, cudaStream_t st) {
  // tuning knob (read once): GRPIC_PD_MINB=4 selects the 126-register build (GRPIC_PD_MA CTAs per
  // SM), anything else the 96-register one (GRPIC_PD_MB); defaults: compacting -> 126, in place -> 96
  static int minb = -1;
  if (minb < 0) { const char* e = getenv("GRPIC_PD_MINB"); minb = e ? atoi(e) : (COMPACT ? 4 : 5); }
  if (ctx->p.geo_iters != 3)
    return launch_push_deposit<GRPIC_PD_MA, COMPACT, 0>(ctx, ptc, dst, offsets, n_alive, f, J, dt, status, st);
  if (minb == 4)
    return launch_push_deposit<GRPIC_PD_MA, COMPACT, 3>(ctx, ptc, dst, offsets, n_alive, f, J, dt, status, st);
  return launch_push_deposit<GRPIC_PD_MB, COMPACT, 3>(ctx, ptc, dst, offsets, n_alive, f, J, dt, status, st);
}

// live particles per 32-particle tile: each thread reads four flags (16 bytes), eight threads
// cover a tile and add their counts by shuffles
__global__ void __launch_bounds__(256) tile_live_kernel(const uint32_t* flag, int64_t n, uint32_t* counts) {
  const int64_t k = ((int64_t)blockIdx.x * 256 + threadIdx.x) * 4;
  uint32_t c = 0;
  if (k + 4 <= n) {
    const uint4 f = *reinterpret_cast<const uint4*>(flag + k);
    c = !(f.x & 2u) + !(f.y & 2u) + !(f.z & 2u) + !(f.w & 2u);
  } else {
    for (int64_t q = k; q < n; ++q) c += !(flag[q] & 2u);
  }
  c += __shfl_xor_sync(0xffffffffu, c, 1);
  c += __shfl_xor_sync(0xffffffffu, c, 2);
  c += __shfl_xor_sync(0xffffffffu, c, 4);
  if ((threadIdx.x & 7) == 0 && k < n) counts[k >> 5] = c;
}
// out[k] for k in [*n_alive, n): flag = removed
__global__ void mark_tail_range_kernel(grpic_particles out, int64_t n, const int64_t* n_alive) {
  for (int64_t k = *n_alive + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n;
       k += (int64_t)gridDim.x * blockDim.x) {
    out.flag[k] = 2u;
    out.cell[k] = 0xFFFFFFFFu;
  }
}

bool ptc_args_ok(const grpic_particles* p) {
  return p && p->n >= 0 && p->x1 && p->x2 && p->x3 && p->u1 && p->u2 && p->u3 && p->w && p->cell && p->flag;
}
bool tma_aligned(const grpic_particles* p) {
  const uintptr_t a = (uintptr_t)p->x1 | (uintptr_t)p->x2 | (uintptr_t)p->x3 | (uintptr_t)p->u1 |
                      (uintptr_t)p->u2 | (uintptr_t)p->u3 | (uintptr_t)p->w | (uintptr_t)p->flag;
  return (a & 15u) == 0;
}
bool grid_args_ok(const grpic_fields* f, const grpic_current* J) {
  return f && J && f->Dr && f->Dth && f->Dph && f->Br && f->Bth && f->Bph && J->Fr && J->Fth && J->Fph;
}

}  // namespace

extern "C" int grpic_push_deposit(grpic_ctx* ctx, grpic_particles* ptc, const grpic_fields* fields,
                                  grpic_current* flux, double dt, uint32_t* status, void* stream) {
  if (!ctx || !ptc_args_ok(ptc) || !grid_args_ok(fields, flux) || !(dt > 0.0)) return GRPIC_ERR_ARG;
  // the particle tiles are fetched with 1-D bulk TMA copies: 16-byte aligned arrays
  if (!tma_aligned(ptc)) return GRPIC_ERR_ARG;
  if (ptc->n == 0) return GRPIC_OK;
  if (ptc->n > 0xFFFFFFF0LL) return GRPIC_ERR_ARG;
  const int rc = dispatch_push_deposit<false>(ctx, *ptc, *ptc, nullptr, nullptr, *fields, *flux, dt, status,
                                              (cudaStream_t)stream);
  grpic_count_launches(1);
  return rc;
}

extern "C" int grpic_push_deposit_compact(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out,
                                          const grpic_fields* fields, grpic_current* flux, double dt,
                                          int64_t* n_alive, uint32_t* status, void* stream) {
  if (!ctx || !in || in->n < 0 || !out || !n_alive || !grid_args_ok(fields, flux) || !(dt > 0.0))
    return GRPIC_ERR_ARG;
  const int64_t n = in->n;
  out->n = n;
  cudaStream_t st = (cudaStream_t)stream;
  if (n == 0) {
    GRPIC_CUDA_OK(cudaMemsetAsync(n_alive, 0, sizeof(int64_t), st));
    return GRPIC_OK;
  }
  if (!ptc_args_ok(in) || !ptc_args_ok(out) || out->x1 == in->x1 || !tma_aligned(in) || n > 0xFFFFFFF0LL)
    return GRPIC_ERR_ARG;
  const size_t ntiles = (size_t)((n + 31) / 32);
  const size_t need = (ntiles + ntiles / 2048 + 4096) * sizeof(uint32_t);
  if (!ctx->ws || ctx->ws_bytes < need) return GRPIC_ERR_WORKSPACE;
  uint32_t* offsets = (uint32_t*)ctx->ws;
  tile_live_kernel<<<(unsigned)((n + 1023) / 1024), 256, 0, st>>>(in->flag, n, offsets);
  int rc = grpic_exclusive_scan(offsets, ntiles, offsets + ntiles, st);
  if (rc != GRPIC_OK) return rc;
  rc = dispatch_push_deposit<true>(ctx, *in, *out, offsets, n_alive, *fields, *flux, dt, status, st);
  if (rc != GRPIC_OK) return rc;
  mark_tail_range_kernel<<<ctx->sm_count, 256, 0, st>>>(*out, n, n_alive);
  grpic_count_launches(3);
  return grpic_launch_ok();
}
