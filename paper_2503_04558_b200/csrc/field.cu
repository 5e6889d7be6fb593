// GR Maxwell field update (Eq.9-11, B8-B11) for sm_100a.
//
// Sweep kernel design: one warp owns 32 consecutive columns (r
// index, the fastest dimension) and MARCHES over a chunk of theta rows.  Per row each lane
//   1. loads the six field values of its own node (coalesced 256-byte row segments),
//   2. computes the 14 metric coefficients of (B9)/(B11) inline from 1-D tables
//      (one rsqrt per staggered location; no coefficient arrays in HBM),
//   3. forms the "coefficient x field" products at the field's own location
//      and exchanges them with its r-neighbours by warp shuffles (B9/B11 average in r only),
//   4. forms the six auxiliary fields, exchanges H_phi,H_theta / E_phi,E_theta with r-neighbours,
//   5. keeps the previous one/two rows of auxiliary fields in registers, so the circulations
//      (B8)/(B10) of row j are complete when row j+1 has been formed,
//   6. applies the predictor (9) or corrector (10) update, axis conditions (Eq.11), radial
//      guard copies and (last sweep) the damping layer in the epilogue.
// No shared memory, no block barrier; lanes 2..29 of each warp produce output (halo 2+2).
#include <math.h>
#include <stdlib.h>

#include "grpic_internal.cuh"

namespace {

constexpr int kOutCols = 28;   // output columns per warp
#ifndef GRPIC_FS_WARPS
#define GRPIC_FS_WARPS 2
#endif
#ifndef GRPIC_FS_STAGES
#define GRPIC_FS_STAGES 2
#endif
constexpr int kWarpsPerBlock = GRPIC_FS_WARPS;
constexpr int kStages = GRPIC_FS_STAGES;   // ring depth of the TMA path (rows in flight per warp)

struct SweepArgs {
  const double* in[6];    // iterate being evaluated (D^r,D^th,D^ph,B^r,B^th,B^ph)
  const double* base[6];  // MODE 0: F^n; MODE 1: F^n + dt (alpha_i C^n - J)
  const double* J[3];     // MODE 0 only (may be null)
  const double* bg[6];    // damping background (last sweep; may be null)
  double* out[6];
  double* base_out[6];    // MODE 0: where to store the corrector base (may be null)
  double dt, a_impl, b_impl;
  int last;               // apply damping
  int prefetch;           // software prefetch into L1 one row ahead
  int tma;                // stream the rows of interior warps through shared memory with bulk TMA copies
  int bcols, nchunks;     // CTA grid: column blocks x row chunks (linearised, edge blocks first)
  int row_chunk;          // output rows per warp (chosen per launch: one full wave of warps)
  int damp_cells;
  double damp_coef;
};

struct Coef {  // at one staggered location
  double q;      // alpha*gamma_rr = sqrt(1+z)
  double al;     // alpha
  double rho2;
  double s;
};
// 1/sqrt(x): MUFU.RSQ64H seed + two Newton steps (~1 ulp), no special-case path
__device__ __forceinline__ double rsqrt_nr(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double h = 0.5 * x;
  double e = fma(-(h * y), y, 0.5);
  y = fma(y, e, y);
  e = fma(-(h * y), y, 0.5);
  return fma(y, e, y);
}
// ---- bulk TMA (cp.async.bulk) + mbarrier plumbing ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
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
  } while (!ok);
}
// one lane of the (converged) warp: the guarded region stays on the uniform datapath
__device__ __forceinline__ bool elect_one() {
  uint32_t p;
  asm volatile("{ .reg .pred P; elect.sync _|P, 0xffffffff; selp.u32 %0, 1, 0, P; }" : "=r"(p));
  return p != 0;
}
// 256-byte bulk copy global -> shared from raw addresses (shared-window destination and barrier)
__device__ __forceinline__ void tma_load_raw(uint32_t dst32, uint64_t src, uint32_t bar32) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], 256, [%2];" ::"r"(dst32),
      "l"(src), "r"(bar32)
      : "memory");
}
__device__ __forceinline__ void prefetch_l1(const double* p) {
  asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
}
__device__ __forceinline__ Coef coef_at(const GridDev& g, double r, double s, double c) {
  Coef k;
  k.rho2 = fma(g.a2 * c, c, r * r);
  const double B = fma(2.0 * g.M, r, k.rho2);
  const double rs = rsqrt_nr(k.rho2 * B);
  k.al = k.rho2 * rs;
  k.q = B * rs;
  k.s = s;
  return k;
}
// alpha*gamma_rphi, sqrt(gamma)*beta^r, alpha*gamma_thth, alpha*gamma_phph
__device__ __forceinline__ double c_rphi(const GridDev& g, const Coef& k) { return -g.a * k.s * k.s * k.q; }
__device__ __forceinline__ double c_sgb(const GridDev& g, const Coef& k, double r) { return 2.0 * g.M * r * k.s * k.al; }
__device__ __forceinline__ double c_thth(const Coef& k) { return k.rho2 * k.al; }
__device__ __forceinline__ double c_phph(const GridDev& g, const Coef& k) {
  const double s2 = k.s * k.s;
  return s2 * fma(g.a2 * s2, k.q, k.rho2 * k.al);
}

__device__ __forceinline__ double shfl_up1(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_dn1(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// MODE 0: predictor (Eq.9) + store corrector base; MODE 1: corrector (Eq.10); MODE 2: write
// the circulations themselves (diagnostics).
// FAST: the warp's 28 output columns and its output rows lie strictly inside the physical
// range of every component (no axis row, no first/last column): every range test, guard copy
// and clamp folds away at compile time.  94 % of the warps of a 2048^2 sweep take this path.
//
// TMA (implies FAST): the warp streams its rows through a private ring of stages in shared
// memory (kStages deep).  A "packet" for iteration jj = the six iterate values of row jj, and the corrector
// base + six area factors of row jj-1 (what that iteration's epilogue reads): 18 segments of
// 32 doubles, each fetched by ONE 256-byte bulk TMA copy issued by lanes 0..17 in parallel and
// signalled on the stage's mbarrier.  Packet jj+kStages is requested as soon as packet jj is
// consumed, so kStages rows are always in flight per warp without holding a register or an L1
// line (measured, field step at 2048^2 / 4096^2: 2 warps x 2 stages per CTA 1.58 / 5.39 ms, 4 x 2
// 1.63 / 5.49, 2 x 3 1.62 / 5.56; deeper rings cost occupancy).
constexpr int kSeg = 18;
template <int MODE, bool FAST, bool TMA>
__device__ __forceinline__ void sweep_rows(const GridDev& g, const SweepArgs& A, int lane, int ibase,
                                           int jstart, int jend, double* ring, uint64_t* bars) {
  const int i = ibase - 2 + lane;                       // this lane's column
  // ---- TMA plumbing.  One elected lane arms the stage's mbarrier and issues the packet's 18 (6 in the
  // first iteration, 12 for the diagnostics mode) bulk copies with warp-uniform addresses.  (Round 1
  // let lanes 0..17 issue one copy each: ptxas serialises such divergent UBLKCP issue in an
  // ELECT / R2UR / BRA.U loop, ~160 of the 613 instructions per row, profiles/r02_final.md.) ----
  // MODE 0 (predictor): the base of row jj-1 IS the iterate of row jj-1, which the previous iteration
  // read: it is carried in registers (Fp) instead of being fetched again, and its six slots of the
  // packet take the three J rows instead (no load is issued from inside the epilogue any more)
  const bool jt = TMA && MODE == 0 && A.J[0] && A.J[1] && A.J[2];
  auto request = [&](int jj, int stage) {               // packet jj -> ring stage
    if (jj > jend) return;
    const bool epi = (jj - 1 >= jstart);                // epilogue operands of row jj-1 wanted
    if (elect_one()) {
      const uint32_t nseg = epi ? (MODE == 1 ? 18u : MODE == 0 ? (jt ? 15u : 12u) : 12u) : 6u;
      const uint32_t bar32 = smem_u32(&bars[stage]);
      const uint32_t dst32 = smem_u32(ring) + (uint32_t)stage * (kSeg * 256u);
      mbar_expect_tx(&bars[stage], nseg * 256u);
      // one byte offset for the six iterate rows (row jj), one for the epilogue operands (row jj-1):
      // every copy is then pointer + offset
      const uint64_t off0 = ((uint64_t)(jj + g.j0) * (uint64_t)g.pitch + (uint64_t)(ibase - 2 + g.i0)) * 8u;
      const uint64_t off1 = off0 - (uint64_t)g.pitch * 8u;
#pragma unroll
      for (int c = 0; c < 6; ++c) tma_load_raw(dst32 + c * 256u, (uint64_t)A.in[c] + off0, bar32);
      if (epi) {
        if (MODE == 1) {
#pragma unroll
          for (int c = 0; c < 6; ++c) tma_load_raw(dst32 + (6 + c) * 256u, (uint64_t)A.base[c] + off1, bar32);
        }
        if (MODE == 0 && jt) {
#pragma unroll
          for (int c = 0; c < 3; ++c) tma_load_raw(dst32 + (6 + c) * 256u, (uint64_t)A.J[c] + off1, bar32);
        }
        tma_load_raw(dst32 + 12 * 256u, (uint64_t)g.iADr + off1, bar32);
        tma_load_raw(dst32 + 13 * 256u, (uint64_t)g.iADth + off1, bar32);
        tma_load_raw(dst32 + 14 * 256u, (uint64_t)g.iADph + off1, bar32);
        tma_load_raw(dst32 + 15 * 256u, (uint64_t)g.iABr + off1, bar32);
        tma_load_raw(dst32 + 16 * 256u, (uint64_t)g.iABth + off1, bar32);
        tma_load_raw(dst32 + 17 * 256u, (uint64_t)g.iABph + off1, bar32);
      }
    }
  };
  if (TMA) {
    if (lane == 0) {
#pragma unroll
      for (int q = 0; q < kStages; ++q) mbar_init(&bars[q], 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
#pragma unroll
    for (int q = 0; q < kStages; ++q) request(jstart - 1 + q, q);
  }
  const int ic = FAST ? i : min(max(i, -g.ng), g.nr + g.ng);       // clamped for loads
  const bool writer = (lane >= 2) && (lane < 2 + kOutCols) && (FAST || i <= g.nr);

  const double r_n = __ldg(g.r_n + ic + g.i0), r_h = __ldg(g.r_h + ic + g.i0);
  const double dr_n = __ldg(g.dr_n + ic + g.i0), dr_h = __ldg(g.dr_h + ic + g.i0);

  // previous rows of auxiliary fields
  double Hph_p = 0, Hph_im1_p = 0, Hr_p = 0, Hth_p = 0, Hth_im1_p = 0;
  double Eph_p = 0, Eph_ip1_p = 0, Er_p = 0, Eth_p = 0, Eth_ip1_p = 0;
  double Hph_pp = 0, Hr_pp = 0;
  double Fp[6] = {0, 0, 0, 0, 0, 0};                    // MODE 0 with TMA: F^n of the previous row

  for (int jj = jstart - 1; jj <= jend; ++jj) {
    // ---- auxiliary fields of row jj ----
    double Hph = 0, Hr = 0, Hth = 0, Eph = 0, Er = 0, Eth = 0;
    const int nit = jj - (jstart - 1);
    const int stg = nit % kStages;
    const double* rs = ring + (stg * kSeg) * 32 + lane;            // this iteration's ring stage
    double Fin[6];
    {
      const size_t k = g.idx(ic, jj);
      if (!TMA && A.prefetch) {
        // A.prefetch rows ahead: the iterate, and the operands of the epilogue (corrector base,
        // area factors) of the row that far ahead
        const int d = A.prefetch;
        const size_t kp = k + (size_t)d * g.pitch;
        if (jj + d <= jend) {
#pragma unroll
          for (int c = 0; c < 6; ++c) prefetch_l1(A.in[c] + kp);
        }
        if (jj + d - 1 >= jstart && jj + d - 1 < jend) {
          const size_t ke = kp - g.pitch;
          if (MODE != 2) {
#pragma unroll
            for (int c = 0; c < 6; ++c) prefetch_l1(A.base[c] + ke);
          }
          prefetch_l1(g.iADr + ke); prefetch_l1(g.iADth + ke); prefetch_l1(g.iADph + ke);
          prefetch_l1(g.iABr + ke); prefetch_l1(g.iABth + ke); prefetch_l1(g.iABph + ke);
        }
      }
      if (TMA) mbar_wait(&bars[stg], (uint32_t)(nit / kStages) & 1u);
      const double Dr = TMA ? rs[0] : __ldg(A.in[0] + k), Dth = TMA ? rs[32] : __ldg(A.in[1] + k);
      const double Dph = TMA ? rs[64] : __ldg(A.in[2] + k), Br = TMA ? rs[96] : __ldg(A.in[3] + k);
      const double Bth = TMA ? rs[128] : __ldg(A.in[4] + k), Bph = TMA ? rs[160] : __ldg(A.in[5] + k);
      Fin[0] = Dr; Fin[1] = Dth; Fin[2] = Dph; Fin[3] = Br; Fin[4] = Bth; Fin[5] = Bph;
      const double sn = __ldg(g.sin_n + jj + g.j0), cn = __ldg(g.cos_n + jj + g.j0);
      const double sh = __ldg(g.sin_h + jj + g.j0), ch = __ldg(g.cos_h + jj + g.j0);
      const Coef knn = coef_at(g, r_n, sn, cn), khn = coef_at(g, r_h, sn, cn);
      const Coef knh = coef_at(g, r_n, sh, ch), khh = coef_at(g, r_h, sh, ch);
      const double P1 = c_rphi(g, khh) * Bph, P6 = c_sgb(g, khh, r_h) * Bph;
      const double P2 = c_sgb(g, knn, r_n) * Dph, P5 = c_rphi(g, knn) * Dph;
      const double P3 = c_rphi(g, knh) * Br, P4 = c_sgb(g, knh, r_n) * Dth;
      const double P7 = c_rphi(g, khn) * Dr, P8 = c_sgb(g, khn, r_h) * Bth;
      const double P1m = shfl_up1(P1), P6m = shfl_up1(P6), P7m = shfl_up1(P7), P8m = shfl_up1(P8);
      const double P2p = shfl_dn1(P2), P5p = shfl_dn1(P5), P3p = shfl_dn1(P3), P4p = shfl_dn1(P4);
      const bool row_n = FAST || ((jj >= 0) && (jj <= g.nth));      // node-in-theta rows
      const bool row_h = FAST || ((jj >= 0) && (jj <= g.nth - 1));  // half-in-theta rows
      if (row_n) {
        Hth = fma(c_thth(khn), Bth, 0.5 * (P2 + P2p));                       // (B9)
        Er = fma(khn.q, Dr, 0.5 * (P5 + P5p));                               // (B11)
        Eph = fma(c_phph(g, knn), Dph, 0.5 * (P7 + P7m) + 0.5 * (P8 + P8m)); // (B11), 1/2 restored
      }
      if (row_h) {
        Hr = fma(knh.q, Br, 0.5 * (P1 + P1m));                               // (B9)
        Hph = fma(c_phph(g, khh), Bph, 0.5 * (P3 + P3p) - 0.5 * (P4 + P4p)); // (B9)
        Eth = fma(c_thth(knh), Dth, -0.5 * (P6 + P6m));                      // (B11)
      }
    }
    const double Hph_im1 = shfl_up1(Hph), Hth_im1 = shfl_up1(Hth);
    const double Eph_ip1 = shfl_dn1(Eph), Eth_ip1 = shfl_dn1(Eth);

    // ---- outputs of row j = jj-1 ----
    const int j = jj - 1;
    if (j >= jstart && writer) {
      const size_t k = g.idx(i, j);
      const bool axis = !FAST && ((j == 0) || (j == g.nth));
      const bool halfrow = FAST || (j < g.nth);
      const bool halfcol = FAST || (i < g.nr);
      double C[6];
      const double aDr = TMA ? rs[12 * 32] : __ldg(g.iADr + k), aDth = TMA ? rs[13 * 32] : __ldg(g.iADth + k);
      const double aDph = TMA ? rs[14 * 32] : __ldg(g.iADph + k), aBr = TMA ? rs[15 * 32] : __ldg(g.iABr + k);
      const double aBth = TMA ? rs[16 * 32] : __ldg(g.iABth + k), aBph = TMA ? rs[17 * 32] : __ldg(g.iABph + k);
      C[0] = (Hph_p - Hph_pp) * aDr;                                                  // (B8), Eq.(11) on the axes
      C[1] = (Hph_im1_p - Hph_p) * aDth;
      C[2] = fma(Hth_p - Hth_im1_p, g.dth, (Hr_pp - Hr_p) * dr_n) * aDph;
      C[3] = -(Eph - Eph_p) * aBr;                                                    // (B10)
      C[4] = -(Eph_p - Eph_ip1_p) * aBth;
      C[5] = -fma(Eth_ip1_p - Eth_p, g.dth, (Er_p - Er) * dr_h) * aBph;
      // physical range of each component
      const bool ok[6] = {halfcol, halfrow, !axis, halfrow, halfcol && !axis, halfcol && halfrow};
      // i of the last physical column of each component (for the radial guard copies)
      const int hi[6] = {g.nr - 1, g.nr, g.nr, g.nr, g.nr - 1, g.nr - 1};
      double lam = 1.0;
      if (A.last && A.damp_cells > 0) {
        const int i0d = g.nr - A.damp_cells;
        if (i > i0d) {
          const double sd = (double)(i - i0d) / (double)(g.nr - i0d);
          lam = 1.0 - A.damp_coef * sd * sd * sd;
        }
      }
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        double v;
        const bool rowok = (c == 1 || c == 3 || c == 5) ? halfrow : true;
        if (MODE == 2) {
          v = ok[c] ? C[c] : 0.0;
        } else if (MODE == 0) {
          const double Fn = TMA ? Fp[c] : __ldg(A.base[c] + k);
          const double Jc = (c < 3 && A.J[c]) ? (jt ? rs[(6 + c) * 32] : __ldg(A.J[c] + k)) : 0.0;
          v = ok[c] ? fma(A.dt, C[c] - Jc, Fn) : 0.0;
          if (A.base_out[c] && rowok && (FAST || i <= hi[c]))
            A.base_out[c][k] = ok[c] ? fma(A.dt, A.a_impl * C[c] - Jc, Fn) : 0.0;
        } else {
          v = ok[c] ? fma(A.dt * A.b_impl, C[c], TMA ? rs[(6 + c) * 32] : __ldg(A.base[c] + k)) : 0.0;
        }
        if (MODE != 2 && lam != 1.0 && ok[c]) {
          const double b = A.bg[c] ? __ldg(A.bg[c] + k) : 0.0;
          v = fma(v - b, lam, b);
        }
        if (rowok && (FAST || i <= hi[c])) {
          A.out[c][k] = v;
          if (MODE != 2 && !FAST) {
            if (i == 0)
              for (int gq = 1; gq <= g.ng; ++gq) A.out[c][k - gq] = v;
            if (i == hi[c])
              for (int gq = 1; gq <= g.nr + g.ng - hi[c]; ++gq) A.out[c][k + gq] = v;
          }
        }
      }
    }
    if (TMA) {                                          // stage consumed: request the packet kStages rows on
      __syncwarp();
      request(jj + kStages, stg);
    }
    // ---- rotate rows ----
    if (MODE == 0 && TMA) {
#pragma unroll
      for (int c = 0; c < 6; ++c) Fp[c] = Fin[c];
    }
    Hph_pp = Hph_p; Hr_pp = Hr_p;
    Hph_p = Hph; Hph_im1_p = Hph_im1; Hr_p = Hr; Hth_p = Hth; Hth_im1_p = Hth_im1;
    Eph_p = Eph; Eph_ip1_p = Eph_ip1; Er_p = Er; Eth_p = Eth; Eth_ip1_p = Eth_ip1;
  }
}

template <int MODE>
__global__ void __launch_bounds__(32 * kWarpsPerBlock)
field_sweep_kernel(const __grid_constant__ GridDev g, const __grid_constant__ SweepArgs A) {
  const int lane = threadIdx.x & 31;
  // CTA order: the two edge column blocks of every row chunk and the two axis row chunks first
  // (their warps take the slower general path), then the interior blocks, so that no slow CTA
  // ends up in the last wave
  int bx, by;
  {
    const int id = blockIdx.x, edge = 2 * A.nchunks, ic = A.bcols - 2, axis = 2 * ic;
    if (A.bcols < 3 || A.nchunks < 3) { bx = id % A.bcols; by = id / A.bcols; }
    else if (id < edge) { bx = (id & 1) ? A.bcols - 1 : 0; by = id >> 1; }
    else if (id < edge + axis) { bx = 1 + (id - edge) % ic; by = ((id - edge) / ic) ? A.nchunks - 1 : 0; }
    else { bx = 1 + (id - edge - axis) % ic; by = 1 + (id - edge - axis) / ic; }
  }
  const int w = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);   // provably warp-uniform
  const int wcol = bx * kWarpsPerBlock + w;
  const int ibase = wcol * kOutCols;
  if (ibase > g.nr) return;
  const int jstart = by * A.row_chunk;
  const int jend = min(jstart + A.row_chunk, g.nth + 1);  // output rows [jstart, jend)
  __shared__ __align__(128) double ring[kWarpsPerBlock][kStages * kSeg * 32];
  __shared__ __align__(8) uint64_t bars[kWarpsPerBlock][kStages];
  const bool fast = (ibase >= 1) && (ibase + kOutCols - 1 <= g.nr - 2) && (jstart >= 1) && (jend <= g.nth);
  if (fast && A.tma) sweep_rows<MODE, true, true>(g, A, lane, ibase, jstart, jend, ring[w], bars[w]);
  else if (fast) sweep_rows<MODE, true, false>(g, A, lane, ibase, jstart, jend, nullptr, nullptr);
  else sweep_rows<MODE, false, false>(g, A, lane, ibase, jstart, jend, nullptr, nullptr);
}

// Axis values, radial guard copies and theta ghost rows by parity (S8) in ONE launch (round 1: three
// kernels run one after the other, twice per field step).  The three rules are applied in the order
// axis -> radial guards -> ghost rows; here every thread composes the rules it depends on instead of
// reading another thread's output, so the roles never read what this launch writes:
//   rows role    (one thread per physical row and component): radial guards = last physical value
//                (PAPER.md:138), which on the axis rows of D^ph and B^th is the axis value 0;
//   columns role (one thread per padded column and component): D^ph = B^th = 0 on the axis nodes
//                (PAPER.md:132), then the theta ghost rows by parity (r, phi components even; theta
//                components odd); in a guard column the source is the last physical value of its row.
__device__ __forceinline__ double* comp(const grpic_fields& f, int c) {
  return c == 0 ? f.Dr : c == 1 ? f.Dth : c == 2 ? f.Dph : c == 3 ? f.Br : c == 4 ? f.Bth : f.Bph;
}
__global__ void __launch_bounds__(128) guards_kernel(const __grid_constant__ GridDev g, const __grid_constant__ grpic_fields f,
                                                     int row_blocks) {
  const int c = blockIdx.y;
  double* X = comp(f, c);
  const int hi = (c == 0 || c == 4 || c == 5) ? g.nr - 1 : g.nr;        // last physical column
  const bool half_t = (c == 1 || c == 3 || c == 5);
  const bool axis0 = (c == 2 || c == 4);                                // vanishes on the axis nodes
  if ((int)blockIdx.x < row_blocks) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int jhi = half_t ? g.nth - 1 : g.nth;
    if (j > jhi) return;
    const bool on_axis = axis0 && (j == 0 || j == g.nth);
    const double lo = on_axis ? 0.0 : X[g.idx(0, j)], up = on_axis ? 0.0 : X[g.idx(hi, j)];
    for (int i = -g.ng; i < 0; ++i) X[g.idx(i, j)] = lo;
    for (int i = hi + 1; i <= g.nr + g.ng; ++i) X[g.idx(i, j)] = up;
  } else {
    const int i = ((int)blockIdx.x - row_blocks) * blockDim.x + threadIdx.x - g.ng;
    if (i > g.nr + g.ng) return;
    if (axis0 && i >= 0 && i <= hi) {
      X[g.idx(i, 0)] = 0.0;
      X[g.idx(i, g.nth)] = 0.0;
    }
    const int is = min(max(i, 0), hi);                                  // source column: the radial guard rule
    const double par = (c == 1 || c == 4) ? -1.0 : 1.0;
    for (int gq = 1; gq <= g.ng; ++gq) {
      if (!half_t) {
        X[g.idx(i, -gq)] = par * X[g.idx(is, gq)];
        X[g.idx(i, g.nth + gq)] = par * X[g.idx(is, g.nth - gq)];
      } else {
        X[g.idx(i, -gq)] = par * X[g.idx(is, gq - 1)];
        X[g.idx(i, g.nth - 1 + gq)] = par * X[g.idx(is, g.nth - gq)];
      }
    }
    if (half_t) X[g.idx(i, g.nth + g.ng)] = par * X[g.idx(is, g.nth - 1 - g.ng)];
  }
}

int fill_guards(const GridDev& g, grpic_fields* f, cudaStream_t st) {
  const int row_blocks = (g.nth + 1 + 127) / 128, col_blocks = (g.nr + 1 + 2 * g.ng + 127) / 128;
  // (programmatic dependent launch of the guards and sweep kernels, griddepcontrol.wait before their
  // first global access, was measured: field step 1.250 ms with, 1.248 ms without at 2048^2, 4.67 / 4.63 ms
  // at 4096^2 -- nothing to hide, not kept)
  guards_kernel<<<dim3(row_blocks + col_blocks, 6), 128, 0, st>>>(g, *f, row_blocks);
  grpic_count_launches(1);
  return grpic_launch_ok();
}

template <int MODE>
int launch_sweep(const grpic_ctx* ctx, SweepArgs A, cudaStream_t st) {
  const GridDev& g = ctx->g;
  const int wcols = (g.nr + 1 + kOutCols - 1) / kOutCols;
  const int bcols = (wcols + kWarpsPerBlock - 1) / kWarpsPerBlock;
  // rows per warp: whole waves of the resident CTAs, at most max_rows rows per chunk (2 halo rows
  // per chunk), at least 8.  Measured after the TMA issue went to one elected lane (field step at
  // 2048^2 / 4096^2, ms): cap 8: 1.363 / 5.02, 12: 1.359 / 5.00, 16: 1.353 / 4.90, 20: 1.351 / 4.87,
  // 32: 1.428 / 4.93, 48: 1.735 (longer chunks lose DRAM page locality and leave fewer CTAs per wave)
  static int per_sm = 0;
  if (per_sm == 0) {
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, field_sweep_kernel<MODE>, 32 * kWarpsPerBlock,
                                                      0) != cudaSuccess || per_sm < 1)
      per_sm = 1;
  }
  static int max_rows = -1;
  if (max_rows < 0) { const char* e = getenv("GRPIC_FS_MAXROWS"); max_rows = e ? atoi(e) : 20; }
  const int resident = ctx->sm_count * per_sm;
  const int nrows = g.nth + 1;
  const int min_chunks = (nrows + max_rows - 1) / max_rows;
  const int waves = (bcols * min_chunks + resident - 1) / resident;        // whole waves of CTAs
  int chunks = waves * resident / bcols;
  if (chunks < min_chunks) chunks = min_chunks;
  int rows = (nrows + chunks - 1) / chunks;
  if (rows < 8) rows = 8;
  A.row_chunk = rows;
  A.bcols = bcols;
  A.nchunks = (g.nth + 1 + rows - 1) / rows;
  field_sweep_kernel<MODE><<<(unsigned)(A.bcols * A.nchunks), 32 * kWarpsPerBlock, 0, st>>>(g, A);
  grpic_count_launches(1);
  return grpic_launch_ok();
}

bool fields_ok(const grpic_fields* f) {
  return f && f->Dr && f->Dth && f->Dph && f->Br && f->Bth && f->Bph;
}
void to_array(const grpic_fields* f, const double* out[6]) {
  out[0] = f->Dr; out[1] = f->Dth; out[2] = f->Dph; out[3] = f->Br; out[4] = f->Bth; out[5] = f->Bph;
}

}  // namespace

extern "C" {

int grpic_fill_guards(grpic_ctx* ctx, grpic_fields* fields, void* stream) {
  if (!ctx || !fields_ok(fields)) return GRPIC_ERR_ARG;
  return fill_guards(ctx->g, fields, (cudaStream_t)stream);
}

int grpic_circulation(grpic_ctx* ctx, const grpic_fields* fields, double* const out[6], void* stream) {
  if (!ctx || !fields_ok(fields) || !out) return GRPIC_ERR_ARG;
  SweepArgs A = {};
  to_array(fields, A.in);
  for (int c = 0; c < 6; ++c) {
    if (!out[c]) return GRPIC_ERR_ARG;
    A.out[c] = out[c];
  }
  return launch_sweep<2>(ctx, A, (cudaStream_t)stream);
}

int grpic_field_step(grpic_ctx* ctx, grpic_fields* fields, const grpic_current* J,
                     const grpic_fields* background, double dt, void* stream) {
  if (!ctx || !fields_ok(fields) || !(dt >= 0.0)) return GRPIC_ERR_ARG;
  if (background && !fields_ok(background)) return GRPIC_ERR_ARG;
  if (J && (!J->Fr || !J->Fth || !J->Fph)) return GRPIC_ERR_ARG;
  const GridDev& g = ctx->g;
  const size_t n2 = g.size();
  if (!ctx->ws || ctx->ws_bytes < 18 * n2 * sizeof(double)) return GRPIC_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  double* ws = (double*)ctx->ws;
  double* base[6];
  double* itA[6];
  double* itB[6];
  for (int c = 0; c < 6; ++c) {
    base[c] = ws + (size_t)c * n2;
    itA[c] = ws + (size_t)(6 + c) * n2;
    itB[c] = ws + (size_t)(12 + c) * n2;
  }
  double* F[6] = {fields->Dr, fields->Dth, fields->Dph, fields->Br, fields->Bth, fields->Bph};
  int rc = fill_guards(g, fields, st);
  if (rc != GRPIC_OK) return rc;
  const int N = ctx->p.field_iters;
  SweepArgs A = {};
  static int pf = -1;
  if (pf < 0) { const char* e = getenv("GRPIC_FS_PREFETCH"); pf = e ? atoi(e) : 1; }
  A.prefetch = pf;
  static int tma = -1;
  if (tma < 0) { const char* e = getenv("GRPIC_FS_TMA"); tma = e ? atoi(e) : 1; }
  A.tma = tma;
  {
    // bulk copies need 16-byte aligned row segments: element i = 0 is 32-byte aligned in arrays that
    // start on a 32-byte boundary (grpic.h); a caller's view that does not takes the load path
    uintptr_t bits = (uintptr_t)ws;
    for (int c = 0; c < 6; ++c) bits |= (uintptr_t)F[c];
    if (J) bits |= (uintptr_t)J->Fr | (uintptr_t)J->Fth | (uintptr_t)J->Fph;
    if (bits & 15u) A.tma = 0;
  }
  A.dt = dt;
  A.b_impl = ctx->p.beta_impl;
  A.a_impl = 1.0 - ctx->p.beta_impl;
  A.damp_cells = ctx->p.damp_cells;
  A.damp_coef = ctx->p.damp_coef;
  if (background) to_array(background, A.bg);
  // predictor, Eq.(9)
  for (int c = 0; c < 6; ++c) {
    A.in[c] = F[c];
    A.base[c] = F[c];
    A.out[c] = itA[c];
    A.base_out[c] = (N > 0) ? base[c] : nullptr;
  }
  if (J) { A.J[0] = J->Fr; A.J[1] = J->Fth; A.J[2] = J->Fph; }
  A.last = (N == 0);
  rc = launch_sweep<0>(ctx, A, st);
  if (rc != GRPIC_OK) return rc;
  if (N == 0) {
    for (int c = 0; c < 6; ++c)
      GRPIC_CUDA_OK(cudaMemcpyAsync(F[c], itA[c], n2 * sizeof(double), cudaMemcpyDeviceToDevice, st));
  }
  // correctors, Eq.(10); the last one writes the caller's arrays
  double** cur = itA;
  double** nxt = itB;
  for (int it = 0; it < N; ++it) {
    const bool last = (it == N - 1);
    for (int c = 0; c < 6; ++c) {
      A.in[c] = cur[c];
      A.base[c] = base[c];
      A.out[c] = last ? F[c] : nxt[c];
      A.base_out[c] = nullptr;
    }
    A.last = last;
    rc = launch_sweep<1>(ctx, A, st);
    if (rc != GRPIC_OK) return rc;
    double** t = cur; cur = nxt; nxt = t;
  }
  return fill_guards(g, fields, st);
}

}  // extern "C"
