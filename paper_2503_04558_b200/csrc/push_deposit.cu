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
// Ablation switches for the cost table in profiles/ (NOT for production: they change the result).
// Build with e.g. GRPIC_NVCC_EXTRA="-DGRPIC_ABL_NO_DEPOSIT" python -m paper_2503_04558_b200.build --force
//   GRPIC_ABL_NO_GATHER   the 24 field loads are replaced by values made from the position
//   GRPIC_ABL_NO_BORIS    the Boris step is skipped
//   GRPIC_ABL_NO_DEPOSIT  no REDs (the deposit arithmetic goes with them)
//   GRPIC_ABL_K=<n>       n corrector iterations instead of the context's K (0..3)
//   GRPIC_ABL_SMEM_DEPOSIT  the 8-21 adds of a particle go to a 3 x 128-double tile in SHARED memory
//                         (atomicAdd on shared doubles) instead of RED.E.ADD.F64 to global memory: the
//                         arithmetic cost of a CTA-owned J tile without its flush and stray handling

// Charge-conserving deposit of one move (Eq.21-23) on the 3x3-node window anchored at the
// lower of the old and new cell in each direction: a move of less than one cell touches at
// most two cells per direction, so 2 F_r faces x 3 rows, 3 columns x 2 F_theta faces and 3x3
// F_phi nodes hold every non-zero flux.  Inputs per direction: the in-cell fractions of the old
// and new position (fa, fb in [0,1)) and which of the window's two cells each lies in (oa, ob in
// {0,1}).  The CIC shapes on the three nodes are then (1-f, f, 0) or (0, 1-f, f): plain selects,
// no max() (a double fmax costs six instructions for its NaN rules).  No per-slot zero test (each
// costs a divergent branch around the atomic); issuing all 21 REDs unconditionally is LSU-bound
// (12.5 ms vs 7.1 ms at 1e8), so the slots that vanish unless a cell face is crossed are grouped.
__device__ __forceinline__ void deposit_local(const PolyTab& pt, const grpic_current& J, uint32_t anchor, uint32_t pitch,
                                              double Q, double vphi, double idt, double fxa, double fya,
                                              double fxb, double fyb, bool oax, bool oay, bool obx,
                                              bool oby, double (*jt)[128] = nullptr) {
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
  const double c3 = vphi * pt.v[kR3], c6 = vphi * pt.v[kSIXTH];
  const double U0 = fma(c3, Tb0, c6 * Ta0), U1 = fma(c3, Tb1, c6 * Ta1), U2 = fma(c3, Tb2, c6 * Ta2);
  const double V0 = fma(c3, Ta0, c6 * Tb0), V1 = fma(c3, Ta1, c6 * Tb1), V2 = fma(c3, Ta2, c6 * Tb2);
#ifdef GRPIC_ABL_SMEM_DEPOSIT
  {
    // same slots, same grouping; slot (row r, column c) of the window -> word (anchor + c + 37 r) mod 128
#define JT(a, r, c) &jt[a][(anchor + (c) + 37u * (r)) & 127u]
    atomicAdd(JT(0, 0, 0), Ay0 * Px0);          atomicAdd(JT(0, 1, 0), Ay1 * Px0);
    atomicAdd(JT(1, 0, 0), Ax0 * Py0);          atomicAdd(JT(1, 0, 1), Ax1 * Py0);
    atomicAdd(JT(2, 0, 0), fma(Sb0, U0, Sa0 * V0));  atomicAdd(JT(2, 0, 1), fma(Sb1, U0, Sa1 * V0));
    atomicAdd(JT(2, 1, 0), fma(Sb0, U1, Sa0 * V1));  atomicAdd(JT(2, 1, 1), fma(Sb1, U1, Sa1 * V1));
    if (cx) {
      atomicAdd(JT(0, 0, 1), Ay0 * Px1);    atomicAdd(JT(0, 1, 1), Ay1 * Px1);
      atomicAdd(JT(1, 0, 2), Ax2 * Py0);
      atomicAdd(JT(2, 0, 2), fma(Sb2, U0, Sa2 * V0));    atomicAdd(JT(2, 1, 2), fma(Sb2, U1, Sa2 * V1));
    }
    if (cy) {
      atomicAdd(JT(0, 2, 0), Ay2 * Px0);
      atomicAdd(JT(1, 1, 0), Ax0 * Py1);  atomicAdd(JT(1, 1, 1), Ax1 * Py1);
      atomicAdd(JT(2, 2, 0), fma(Sb0, U2, Sa0 * V2));   atomicAdd(JT(2, 2, 1), fma(Sb1, U2, Sa1 * V2));
      if (cx) {
        atomicAdd(JT(0, 2, 1), Ay2 * Px1);
        atomicAdd(JT(1, 1, 2), Ax2 * Py1);
        atomicAdd(JT(2, 2, 2), fma(Sb2, U2, Sa2 * V2));
      }
    }
#undef JT
    (void)J; (void)pitch;
    return;
  }
#endif
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

// ---- TMA (cp.async.bulk) + mbarrier plumbing for the per-warp particle tile rings ----
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
// try_wait suspends the warp in hardware up to a system time limit before it returns false: no
// sleep loop around it (r02a: the NANOSLEEP version executed 14 sleeps + 15 polls per warp tile).
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{ .reg .pred p;\n"
      "W: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@!p bra W; }" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
// one lane of the (converged) warp: the compiler keeps the guarded region on the uniform datapath
__device__ __forceinline__ bool elect_one() {
  uint32_t p;
  asm volatile("{ .reg .pred P; elect.sync _|P, 0xffffffff; selp.u32 %0, 1, 0, P; }" : "=r"(p));
  return p != 0;
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

// One warp tile of particle input staged in shared memory: structure of arrays, kWTile = 64
// particles = two 32-particle halves that the warp pushes one after the other (eight 512-byte
// bulk copies per 64 particles: the issue cost of the staging is halved against 32-particle tiles).
constexpr int kWarps = kBlock / 32;
constexpr int kWTile = 64;
#ifndef GRPIC_PD_STAGES
#define GRPIC_PD_STAGES 2
#endif
constexpr int kPdStages = GRPIC_PD_STAGES;   // particle tiles in flight per warp
struct __align__(128) WTile {
  double x1[kWTile], x2[kWTile], x3[kWTile], u1[kWTile], u2[kWTile], u3[kWTile], w[kWTile];
  uint32_t flag[kWTile];   // bits 0-2: species / removed; COMPACT parks the lane's output rank in bits 8-13
};
constexpr uint32_t kTileBytes = 7u * kWTile * 8u + kWTile * 4u;

// Persistent kernel, warp-autonomous.  Warp w of the grid walks the 64-particle tiles w, w + W,
// w + 2W, ... (W = warps in the grid) through its OWN ring of kPdStages shared-memory stages, each
// filled by eight 1-D bulk TMA copies signalled on the stage's mbarrier.  No block barrier and no
// coupling between the warps of a CTA: a warp waits only for its own data, which was requested
// kPdStages - 1 tile times (~10 us) earlier.  Stage hand-back (write-after-read): every lane's
// shared-memory reads of a stage feed values it has consumed before the __syncwarp() that precedes
// the refill, __syncwarp() orders the lanes' accesses, and only then does the elected lane issue
// the bulk copies into that stage (the per-stage "empty" barrier of the usual TMA pipeline,
// collapsed to a warp barrier because producer and consumers are the same warp).  The last,
// partial tile (n % 64 != 0) is staged with plain loads.
//
// COMPACT: the results are stored to `dst` at offsets[32-particle tile] + rank among the tile's
// live lanes (offsets = exclusive scan of the per-tile live counts of `ptc`), i.e. particles
// already flagged removed are squeezed out on the way, order preserved; the weight travels along.
// Otherwise dst == ptc and the update is in place.
// registers per thread for MINB resident 64-thread CTAs: 8 -> 128, 9 -> 112, 10 -> 96 (ptxas left to
// itself picks 96 for MINB = 9)
constexpr int pd_max_regs(int minb) { return minb <= 8 ? 128 : (minb == 9 ? 112 : 96); }
template <int MINB, bool COMPACT, int KT, bool TAB, bool VAY = false>
__global__ void __launch_bounds__(kBlock) __maxnreg__(pd_max_regs(MINB))
push_deposit_kernel(const __grid_constant__ GridDev g, const __grid_constant__ grpic_particles ptc,
                    const __grid_constant__ grpic_particles dst, const uint32_t* __restrict__ offsets,
                    const __grid_constant__ grpic_fields f, const __grid_constant__ grpic_current J,
                    const __grid_constant__ PolyTab pt, double dt, int K, uint32_t* status,
                    unsigned long long* removed, unsigned long long* clock_probe) {
  // SM clock during this launch (grpic_set_clock_probe): the first thread of the persistent grid notes
  // the SM cycle counter and the nanosecond timer when it starts and when it has pushed its last tile
  const bool probe = clock_probe && blockIdx.x == 0 && threadIdx.x == 0;
  if (probe) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    clock_probe[0] = (unsigned long long)clock64();
    clock_probe[1] = t;
  }
  __shared__ WTile tiles[kWarps][kPdStages];
  __shared__ __align__(8) uint64_t full[kWarps][kPdStages];
  // COMPACT: the aligned 16 bytes of `offsets` that hold each staged tile's two output offsets.
  // Shared memory is kept below 15872 bytes per CTA on purpose: 8 CTAs then fit the 132 KB carve-out
  // and leave 124 KB of L1 to the gather (the 164 KB carve-out a few bytes more would select: 92 KB).
  __shared__ __align__(16) uint32_t sob[COMPACT ? kWarps : 1][COMPACT ? kPdStages : 1][4];
#ifdef GRPIC_ABL_SMEM_DEPOSIT
  __shared__ double jtile[3][128];
  for (int q = threadIdx.x; q < 3 * 128; q += kBlock) (&jtile[0][0])[q] = 0.0;
  __syncthreads();
#endif
  uint32_t tid_x;
  asm volatile("mov.u32 %0, %%tid.x;" : "=r"(tid_x));
  const uint32_t lane = tid_x & 31u;
  const uint32_t warp = __shfl_sync(0xffffffffu, tid_x >> 5, 0);   // provably warp-uniform
  // all particle indices fit 32 bits (the C entry rejects n > 0xFFFFFFF0): one-instruction addressing
  const uint32_t n32 = (uint32_t)ptc.n;
  const uint32_t ntiles = (n32 + kWTile - 1) / kWTile;
  const uint32_t wstride = gridDim.x * kWarps;
  const uint32_t wtile0 = blockIdx.x * kWarps + warp;
  const double idt = 1.0 / dt;
  WTile* const ring = tiles[warp];
  uint64_t* const bars = full[warp];

  const uint64_t stream_policy = l2_evict_first_policy();
  auto issue = [&](uint32_t tile, int stage) {      // whole warp, converged; full tiles only
    const uint32_t k0 = tile * kWTile;
    if (tile >= ntiles || k0 + kWTile > n32) return;
    if (elect_one()) {
      WTile& T = ring[stage];
      uint64_t* bar = &bars[stage];
      mbar_expect_tx(bar, kTileBytes + (COMPACT ? 16u : 0u));
      // the tile's two output offsets ride along (offsets[2 tile], [2 tile + 1], inside an aligned 16 bytes)
      if (COMPACT) tma_load_1d(sob[warp][stage], offsets + ((2u * tile) & ~3u), 16, bar, stream_policy);
      tma_load_1d(T.x1, ptc.x1 + k0, kWTile * 8, bar, stream_policy);
      tma_load_1d(T.x2, ptc.x2 + k0, kWTile * 8, bar, stream_policy);
      tma_load_1d(T.x3, ptc.x3 + k0, kWTile * 8, bar, stream_policy);
      tma_load_1d(T.u1, ptc.u1 + k0, kWTile * 8, bar, stream_policy);
      tma_load_1d(T.u2, ptc.u2 + k0, kWTile * 8, bar, stream_policy);
      tma_load_1d(T.u3, ptc.u3 + k0, kWTile * 8, bar, stream_policy);
      tma_load_1d(T.w, ptc.w + k0, kWTile * 8, bar, stream_policy);
      tma_load_1d(T.flag, ptc.flag + k0, kWTile * 4, bar, stream_policy);
    }
  };
  if (elect_one()) {
#pragma unroll
    for (int q = 0; q < kPdStages; ++q) mbar_init(&bars[q], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();
#pragma unroll
  for (int q = 0; q < kPdStages; ++q) issue(wtile0 + q * wstride, q);

  // one loop iteration = one 32-particle half of the warp's current 64-particle tile
  uint32_t tile = wtile0;
  for (uint32_t j = 0; tile < ntiles; ++j) {
  const uint32_t half = j & 1u, it = j >> 1;
  const uint32_t stage = it % kPdStages;
  WTile& T = ring[stage];
  if (half == 0) {
    if (tile * kWTile + kWTile <= n32) {
      mbar_wait(&bars[stage], (it / kPdStages) & 1u);
    } else {                                        // partial last tile: every lane stages its own slots
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const uint32_t s2 = h * 32 + lane, k = tile * kWTile + s2;
        if (k < n32) {
          T.x1[s2] = ptc.x1[k]; T.x2[s2] = ptc.x2[k]; T.x3[s2] = ptc.x3[k];
          T.u1[s2] = ptc.u1[k]; T.u2[s2] = ptc.u2[k]; T.u3[s2] = ptc.u3[k];
          T.w[s2] = ptc.w[k];
          T.flag[s2] = ptc.flag[k];
        } else {
          T.flag[s2] = 2u;
        }
      }
      if (COMPACT && lane < 4) sob[warp][stage][lane] = offsets[((2u * tile) & ~3u) + lane];
      __syncwarp();
    }
    if (COMPACT) {
      // rank of each particle among the live lanes of its 32-particle half, parked in the spare bits
      // of its flag word in shared memory instead of a register that would live across the whole push
      uint32_t lt;
      asm("mov.u32 %0, %%lanemask_lt;" : "=r"(lt));
      const uint32_t f0 = T.flag[lane], f1 = T.flag[32 + lane];
      const uint32_t live0 = __ballot_sync(0xffffffffu, !(f0 & 2u));
      const uint32_t live1 = __ballot_sync(0xffffffffu, !(f1 & 2u));
      T.flag[lane] = (f0 & 7u) | (__popc(live0 & lt) << 8);
      T.flag[32 + lane] = (f1 & 7u) | (__popc(live1 & lt) << 8);
    }
  }

  {
  const uint32_t sl = half * 32 + lane;
  const uint32_t flag_word = T.flag[sl];
  const uint32_t flag = COMPACT ? (flag_word & 7u) : flag_word;
  if (!(flag & 2u)) {
    const double x1 = T.x1[sl], x2 = T.x2[sl];
    // species: charge sign of e-/e+; a photon (bit2) feels no Lorentz force
    // (sgn = 0 makes the Boris step the exact identity), has eps = 0 and carries no charge
    const bool photon = (flag & 4u) != 0;
    const double sgn = photon ? 0.0 : ((flag & 1u) ? 1.0 : -1.0);

    // ---- gather (first order, each component from its own staggered lattice): the 24
    // loads are issued first, exp / sincos / metric run while they are in flight ----
    const double xa = (x1 - g.xi_in) * g.inv_dxi, ya = x2 * g.inv_dth;
    const double fin = floor(xa), fjn = floor(ya);
    int ia = (int)fin, ja = (int)fjn;
    // a caller bug (an active particle outside [xi_in, xi_out) x [0, pi]) must not become an
    // out-of-bounds access: the cell is clamped, the particle flagged removed, nothing deposited
    const bool offgrid = (uint32_t)ia >= (uint32_t)g.nr || (uint32_t)ja > (uint32_t)g.nth;
    ia = (int)min((uint32_t)ia, (uint32_t)(g.nr - 1));
    ja = (int)min((uint32_t)ja, (uint32_t)g.nth);
    const double fih = floor(xa - 0.5), fjh = floor(ya - 0.5);
    const int ih = offgrid ? ia : (int)fih, jh = offgrid ? ja : (int)fjh;
    const uint32_t bnn = (uint32_t)g.idx(ia, ja), bhn = (uint32_t)g.idx(ih, ja);
    const uint32_t bnh = (uint32_t)g.idx(ia, jh), bhh = (uint32_t)g.idx(ih, jh);
    double G[6][4];
    {
      const double* F6[6] = {f.Dr, f.Dth, f.Dph, f.Br, f.Bth, f.Bph};
      const uint32_t b6[6] = {bhn, bnh, bnn, bnh, bhn, bhh};
#pragma unroll
      for (int c = 0; c < 6; ++c) {
#ifdef GRPIC_ABL_NO_GATHER
        G[c][0] = x1 * (c + 1); G[c][1] = x2 + c; G[c][2] = x1 - c; G[c][3] = x2 * (c + 2);
        (void)F6; (void)b6;
#else
        G[c][0] = __ldg(F6[c] + b6[c]);
        G[c][1] = __ldg(F6[c] + b6[c] + 1);
        G[c][2] = __ldg(F6[c] + b6[c] + g.pitch);
        G[c][3] = __ldg(F6[c] + b6[c] + g.pitch + 1);
#endif
      }
    }

    // ---- r, sin, cos at x^n.  TAB (cells no larger than kSmallStep in xi and theta, i.e. grids of
    // ~1000 cells and more): from the node tables r_i = exp(xi_i), sin(theta_j), cos(theta_j) that
    // the field solver uses, times the short series of the in-cell offset; else the full exp / sincos
    double r0, s0, c0;
    if (TAB) {
      const double rn = __ldg(g.r_n + (ia + g.i0));
      const double sn = __ldg(g.sin_n + (ja + g.j0)), cn = __ldg(g.cos_n + (ja + g.j0));
      r0 = fma(rn, expm1_small(pt, x1 - fma(fin, g.dxi, g.xi_in)), rn);
      sincos_shift(pt, sn, cn, x2 - fjn * g.dth, s0, c0);
    } else {
      r0 = exp_pt(pt, x1);
      sincos_pt(pt, x2, s0, c0);
    }
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
    double ur = T.u1[sl], ut = T.u2[sl], up = T.u3[sl];
#ifndef GRPIC_ABL_NO_BORIS
    if (VAY) vay(g, p0, alpha0, sgn, dt, D, B, ur, ut, up);      // PAPER.md:204, grpic_push_deposit_variant
    else boris(g, p0, alpha0, sgn, dt, D, B, ur, ut, up);
#else
    ur += 1e-300 * (D[0] + D[1] + D[2] + B[0] + B[1] + B[2]);     // keeps the gather alive
#endif

    // ---- geodesic predictor + K correctors (Eq.14, 15) ----
    double Xr0, Xt0, Xp0, Ur0, Ut0;
    geodesic_rhs(g, p0, photon ? 0.0 : p0.zp1, ur, ut, up, Xr0, Xt0, Xp0, Ur0, Ut0);
    double dr = Xr0 * dt, dth = Xt0 * dt, dph = Xp0 * dt;      // increments from x^n
    double vr = fma(Ur0, dt, ur), vt = fma(Ut0, dt, ut);
    const double hdt = 0.5 * dt;
#ifdef GRPIC_ABL_K
    const int KK = GRPIC_ABL_K;
    (void)K;
#else
    const int KK = KT > 0 ? KT : K;                 // KT: compile-time corrector count (unrolled)
#endif
#pragma unroll
    for (int ci = 0; ci < KK; ++ci) {
      double s, c;
      // TAB: |dtheta| = dt |X^theta| <= dt alpha / rho <= dt / r < kSmallStep is guaranteed by the dispatch
      if (TAB || fabs(dth) <= kSmallStep) sincos_shift(pt, s0, c0, dth, s, c);
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
    const double r = r0 + dr, ph = T.x3[sl] + dph;
    const double th_dep = x2 + dth;                 // un-reflected new theta: what the deposit sees

    // ---- new logical position: ln r = x1 + 2 atanh(dr / (2 r0 + dr)) ----
    double x1n;
    {
      const double wq = dr * rcp_nr(r0 + r);       // TAB: |dr| <= dt << r, the series always applies
      if (TAB || fabs(wq) <= 0.03) {
        const double w2 = wq * wq;
        double pl = fma(w2, pt.v[kR11], pt.v[kR9]);
        pl = fma(pl, w2, pt.v[kR7]);
        pl = fma(pl, w2, pt.v[kR5]);
        pl = fma(pl, w2, pt.v[kR3]);
        const double at = fma(pl * w2, wq, wq);
        x1n = fma(2.0, at, x1);
      } else {
        x1n = log(r);
      }
    }
    // ---- reflection at the axes: theta -> -theta or 2 pi - theta, u_theta flips ----
    double th = fabs(th_dep);
    // sign bit of th_dep moves into u_theta (th_dep < 0 flips it)
    vt = __hiloint2double(__double2hiint(vt) ^ (__double2hiint(th_dep) & 0x80000000), __double2loint(vt));
    bool reflected = __double2hiint(th_dep) < 0;
    if (th > pt.v[kPI]) { th = pt.v[kTWOPI] - th; vt = -vt; reflected = true; }
    // ---- new position in index space.  The deposit takes the PRODUCT form (x - xi_in) * (1/dxi): it
    // is the expression the next step (and the rho deposit) applies to the stored position, so the
    // charge a particle leaves at its new position is exactly the charge it starts from.  The cell
    // index is the floor of the correctly rounded QUOTIENT (the oracle's division): the product
    // refined by one residual step, q + (a - q d)(1/d), equals the IEEE division whenever 1/d is
    // correctly rounded, which the host guarantees ----
    const double ax = x1n - g.xi_in;
    const double xb = ax * g.inv_dxi, yb = th_dep * g.inv_dth;
    const double fib = floor(xb), fjb = floor(yb);
    const int ib = (int)fib, jb = (int)fjb;
    const double fxb = xb - fib, fyb = yb - fjb;
    const int icq = (int)floor(fma(fma(-xb, g.dxi, ax), g.inv_dxi, xb));
    const int jcq = (int)floor(fma(fma(-yb, g.dth, th_dep), g.inv_dth, yb));
    // finite test on the three quantities that reach the grid (a non-finite momentum alone shows
    // up in the position one step later): the high words, read as floats, are finite floats
    // unless the double is inf / nan or >= 2^1017
    const bool finite = fabsf(__int_as_float(__double2hiint(x1n))) + fabsf(__int_as_float(__double2hiint(th_dep))) +
                            fabsf(__int_as_float(__double2hiint(dph))) < __int_as_float(0x7f800000);
    const bool out = !(x1n >= g.xi_in && x1n < g.xi_out) || offgrid || !finite;
    uint32_t nflag = flag, ncell;
    if (out) {
      nflag |= 2u;
      ncell = 0xFFFFFFFFu;
      if (removed) atomicAdd(removed, 1ull);        // rare (a particle leaves once): lazy-removal bookkeeping
      if (status && (!finite || offgrid))
        atomicOr(status, offgrid ? GRPIC_STATUS_OFFGRID : GRPIC_STATUS_NONFINITE);
    } else {
      int jc = jcq;
      if (reflected) {                              // at an axis: the cell of the mirrored theta
        double yc = th * g.inv_dth;
        yc = fma(fma(-yc, g.dth, th), g.inv_dth, yc);
        jc = (int)floor(yc);
      }
      const int ic = min(max(icq, 0), g.nr - 1);
      jc = min(max(jc, 0), g.nth - 1);
      ncell = (uint32_t)(jc * g.nr + ic);
    }
    // COMPACT: output index = offsets[this 32-particle half] + rank among its live lanes
    const uint32_t kd = COMPACT ? sob[warp][stage][(tile & 1u) * 2u + half] + (T.flag[sl] >> 8) : tile * kWTile + sl;
    __stcs(dst.x1 + kd, x1n); __stcs(dst.x2 + kd, th); __stcs(dst.x3 + kd, ph);   // streaming stores
    __stcs(dst.u1 + kd, vr); __stcs(dst.u2 + kd, vt); __stcs(dst.u3 + kd, up);
    if (COMPACT) __stcs(dst.w + kd, T.w[sl]);
    __stcs(dst.cell + kd, ncell);
    __stcs(dst.flag + kd, nflag);

    // ---- deposit: 3x3 window anchored at the lower of the old / new cell ----
#ifdef GRPIC_ABL_NO_DEPOSIT
    if (false) {
#else
    if (finite && !photon && !offgrid) {
#endif
      const double q = sgn * T.w[sl];
      const double vph = q * dph * idt;
      const int di = ib - ia, dj = jb - ja;
      if ((uint32_t)(di + 1) <= 2u && (uint32_t)(dj + 1) <= 2u) {
        const int iw = min(ia, ib), jw = min(ja, jb);
#ifdef GRPIC_ABL_SMEM_DEPOSIT
        deposit_local(pt, J, (uint32_t)g.idx(iw, jw), (uint32_t)g.pitch, q, vph, idt, xa - fin, ya - fjn, fxb,
                      fyb, ia != iw, ja != jw, ib != iw, jb != jw, jtile);
#else
        deposit_local(pt, J, (uint32_t)g.idx(iw, jw), (uint32_t)g.pitch, q, vph, idt, xa - fin, ya - fjn, fxb,
                      fyb, ia != iw, ja != jw, ib != iw, jb != jw);
#endif
      } else {
        deposit_far(&g, q, idt, vph, xa, xb, ya, yb, J.Fr, J.Fth, J.Fph, status);
      }
    }
  }
  }
  if (half == 1) {       // this warp is done with the stage: refill it with the tile kPdStages steps ahead
    __syncwarp();
    issue(tile + kPdStages * wstride, stage);
    tile += wstride;
  }
  }
#ifdef GRPIC_ABL_SMEM_DEPOSIT
  __syncthreads();      // the tile's content goes somewhere, so that the adds above are not dead code
  for (int q = threadIdx.x; q < 3 * 128; q += kBlock) atomicAdd(J.Fr + q, (&jtile[0][0])[q] * 1e-300);
#endif
  if (probe) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    clock_probe[2] = (unsigned long long)clock64();
    clock_probe[3] = t;
  }
}

template <int MINB, bool COMPACT, int KT, bool TAB, bool VAY = false>
int launch_push_deposit(const grpic_ctx* ctx, const grpic_particles& ptc, const grpic_particles& dst,
                        const uint32_t* offsets, const grpic_fields& f,
                        const grpic_current& J, double dt, uint32_t* status, cudaStream_t st) {
  static int per_sm = 0;   // resident CTAs per SM of this instantiation
  if (per_sm == 0) {
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, push_deposit_kernel<MINB, COMPACT, KT, TAB, VAY>,
                                                      kBlock, 0) != cudaSuccess || per_sm < 1)
      per_sm = 1;
  }
  const int64_t nblocks = (ptc.n + kWarps * kWTile - 1) / (kWarps * kWTile);
  const int64_t resident = (int64_t)ctx->sm_count * per_sm;
  const unsigned grid = (unsigned)(nblocks < resident ? nblocks : resident);
  push_deposit_kernel<MINB, COMPACT, KT, TAB, VAY><<<grid, kBlock, 0, st>>>(ctx->g, ptc, dst, offsets, f, J, kPolyTabHost, dt,
                                                                  ctx->p.geo_iters, status, ctx->removed_counter,
                                                                  ctx->clock_probe);
  return grpic_launch_ok();
}

template <bool COMPACT>
int dispatch_push_deposit(const grpic_ctx* ctx, const grpic_particles& ptc, const grpic_particles& dst,
                          const uint32_t* offsets, const grpic_fields& f,
                          const grpic_current& J, double dt, uint32_t* status, cudaStream_t st) {
  // tuning knob (read once): GRPIC_PD_MINB = resident 64-thread CTAs per SM the kernel is built for:
  // 8 (<= 128 registers, no spills: the default; 5.70 ms per push averaged over a 20-step sort period at
  // 1e8 particles), 9 (<= 112: 5.90 ms) or 10 (<= 96: 5.99 ms) -- profiles/r02h
  static int minb = -1;
  if (minb < 0) { const char* e = getenv("GRPIC_PD_MINB"); minb = e ? atoi(e) : 8; }
  // TAB: cells small enough for the node-table + in-cell series form of r, sin, cos (push_math.cuh),
  // and a time step whose moves |dtheta| <= dt / r, |dr| <= dt stay inside the short series of the
  // correctors and of ln r without a test (r >= r_in - dt during the iterations; factor 2 of margin)
  const bool tab = ctx->g.dxi <= kSmallStep && ctx->g.dth <= kSmallStep && 2.0 * dt <= kSmallStep * exp(ctx->g.xi_in);
  if (ctx->p.geo_iters != 3)
    return launch_push_deposit<GRPIC_PD_MA, COMPACT, 0, false>(ctx, ptc, dst, offsets, f, J, dt, status, st);
  if (!tab)
    return launch_push_deposit<GRPIC_PD_MA, COMPACT, 3, false>(ctx, ptc, dst, offsets, f, J, dt, status, st);
  if (minb <= 8)
    return launch_push_deposit<GRPIC_PD_MA, COMPACT, 3, true>(ctx, ptc, dst, offsets, f, J, dt, status, st);
  if (minb == 9)
    return launch_push_deposit<9, COMPACT, 3, true>(ctx, ptc, dst, offsets, f, J, dt, status, st);
  return launch_push_deposit<GRPIC_PD_MB, COMPACT, 3, true>(ctx, ptc, dst, offsets, f, J, dt, status, st);
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
// survivor count = offsets[last 32-particle tile] + its live lanes (every CTA recomputes it from the
// input flags; CTA 0 publishes it), then out[k] for k in [n_alive, n): flag = removed
__global__ void __launch_bounds__(256) finish_compact_kernel(grpic_particles out, const uint32_t* in_flag, int64_t n,
                                                             const uint32_t* offsets, int64_t* n_alive) {
  __shared__ int64_t na_s;
  if (threadIdx.x < 32) {
    const int64_t last = (n - 1) >> 5, k = last * 32 + threadIdx.x;
    const uint32_t live = __ballot_sync(0xffffffffu, k < n && !(in_flag[k] & 2u));
    if (threadIdx.x == 0) {
      na_s = (int64_t)offsets[last] + __popc(live);
      if (blockIdx.x == 0) *n_alive = na_s;
    }
  }
  __syncthreads();
  for (int64_t k = na_s + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n;
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
  const int rc = dispatch_push_deposit<false>(ctx, *ptc, *ptc, nullptr, *fields, *flux, dt, status,
                                              (cudaStream_t)stream);
  grpic_count_launches(1);
  return rc;
}

// First-order shape with the Vay pusher through the tuned kernel (grpic_push_deposit_variant(1, 1));
// GRPIC_ERR_ARG when the arrays do not allow the bulk-TMA tiles (the caller then takes the general kernel).
int grpic_push_deposit_cic_vay(grpic_ctx* ctx, grpic_particles* ptc, const grpic_fields* fields, grpic_current* flux,
                               double dt, uint32_t* status, cudaStream_t st) {
  if (!ctx || !ptc_args_ok(ptc) || !grid_args_ok(fields, flux) || !(dt > 0.0) || !tma_aligned(ptc) ||
      ptc->n > 0xFFFFFFF0LL)
    return GRPIC_ERR_ARG;
  if (ptc->n == 0) return GRPIC_OK;
  const bool tab = ctx->g.dxi <= kSmallStep && ctx->g.dth <= kSmallStep && 2.0 * dt <= kSmallStep * exp(ctx->g.xi_in);
  grpic_count_launches(1);
  if (ctx->p.geo_iters != 3)
    return launch_push_deposit<GRPIC_PD_MA, false, 0, false, true>(ctx, *ptc, *ptc, nullptr, *fields, *flux, dt, status, st);
  if (!tab)
    return launch_push_deposit<GRPIC_PD_MA, false, 3, false, true>(ctx, *ptc, *ptc, nullptr, *fields, *flux, dt, status, st);
  return launch_push_deposit<GRPIC_PD_MA, false, 3, true, true>(ctx, *ptc, *ptc, nullptr, *fields, *flux, dt, status, st);
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
  rc = dispatch_push_deposit<true>(ctx, *in, *out, offsets, *fields, *flux, dt, status, st);
  if (rc != GRPIC_OK) return rc;
  finish_compact_kernel<<<ctx->sm_count, 256, 0, st>>>(*out, in->flag, n, offsets, n_alive);
  grpic_count_launches(3);
  return grpic_launch_ok();
}
