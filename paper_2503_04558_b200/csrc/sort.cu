// Particle cell-sort (stable LSD radix sort on the cell key) and order-preserving compaction
// of removed particles, with warp-level match/ballot ranking.  Hand-written for sm_100a; no
// CUB/Thrust.  Sort is not part of the paper (BASELINE.json north_star); removal follows
// PAPER.md:138,:364.
#include <stdlib.h>

#include <mutex>

#include "grpic_internal.cuh"

// Scratch of grpic_compact_static: per-tile alive counts + the words of their scan, for at most
// GRPIC_COMPACT_STATIC_MAX_PARTICLES particles (2^26 -> 32768 tiles of 2048 + 16 + 4096 words; 160 KiB
// that every GPU that loads the library holds until exit).  In HOST code this name is a stand-in, not
// a device address: static_scratch() below resolves it with cudaGetSymbolAddress once per device.
constexpr size_t kStaticScratchWords = 40960;
static __device__ __align__(256) uint32_t g_compact_static_scratch[kStaticScratchWords];

namespace {

constexpr int kTile = 2048;     // keys per block
constexpr int kThreads = 256;   // 8 warps, each owns 256 consecutive keys = 8 groups of 32
constexpr int kGroups = 8;
constexpr int kRadix = 256;

// ------------------------------------------------------------------ device-wide exclusive scan
constexpr int kScanTile = 2048;
__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += t;
  }
  return v;
}
// exclusive scan of one 2048-element tile held 8 per thread (blocked); returns tile total
__device__ __forceinline__ uint32_t block_excl_scan8(uint32_t v[8], uint32_t* smem /*>=9*/) {
  uint32_t sum = 0;
#pragma unroll
  for (int m = 0; m < 8; ++m) sum += v[m];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t incl = warp_incl_scan(sum, lane);
  if (lane == 31) smem[w] = incl;
  __syncthreads();
  if (w == 0) {
    const uint32_t ws = (lane < 8) ? smem[lane] : 0u;
    const uint32_t wi = warp_incl_scan(ws, lane);
    if (lane < 8) smem[lane] = wi - ws;
    if (lane == 7) smem[8] = wi;
  }
  __syncthreads();
  uint32_t run = smem[w] + incl - sum;
#pragma unroll
  for (int m = 0; m < 8; ++m) {
    const uint32_t t = v[m];
    v[m] = run;
    run += t;
  }
  return smem[8];
}
// eight consecutive words of one thread: two 16-byte accesses when the array is 16-byte aligned and
// all eight are inside, else word by word (zeros beyond n)
__device__ __forceinline__ void load8(const uint32_t* data, size_t base, size_t n, uint32_t v[8]) {
  if (base + 8 <= n && (((uintptr_t)data) & 15u) == 0) {
    const uint4 a = *reinterpret_cast<const uint4*>(data + base), b = *reinterpret_cast<const uint4*>(data + base + 4);
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
  } else {
#pragma unroll
    for (int m = 0; m < 8; ++m) v[m] = (base + m < n) ? data[base + m] : 0u;
  }
}
__device__ __forceinline__ void store8(uint32_t* data, size_t base, size_t n, const uint32_t v[8]) {
  if (base + 8 <= n && (((uintptr_t)data) & 15u) == 0) {
    *reinterpret_cast<uint4*>(data + base) = make_uint4(v[0], v[1], v[2], v[3]);
    *reinterpret_cast<uint4*>(data + base + 4) = make_uint4(v[4], v[5], v[6], v[7]);
  } else {
#pragma unroll
    for (int m = 0; m < 8; ++m)
      if (base + m < n) data[base + m] = v[m];
  }
}
// sums[b] = sum of tile b (read only)
__global__ void __launch_bounds__(kThreads) tile_sums_kernel(const uint32_t* data, size_t n, uint32_t* sums) {
  __shared__ uint32_t sm[kThreads / 32];
  const size_t base = (size_t)blockIdx.x * kScanTile + (size_t)threadIdx.x * 8;
  uint32_t v[8];
  load8(data, base, n, v);
  uint32_t t = 0;
#pragma unroll
  for (int m = 0; m < 8; ++m) t += v[m];
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) t += __shfl_xor_sync(0xffffffffu, t, d);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = t;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t tot = 0;
    for (int q = 0; q < kThreads / 32; ++q) tot += sm[q];
    sums[blockIdx.x] = tot;
  }
}
// exclusive scan of every tile in place, plus the tile's offset offs[b] (nullable)
__global__ void __launch_bounds__(kThreads) scan_tiles_kernel(uint32_t* data, size_t n, const uint32_t* offs) {
  __shared__ uint32_t sm[9];
  const size_t base = (size_t)blockIdx.x * kScanTile + (size_t)threadIdx.x * 8;
  const uint32_t off = offs ? offs[blockIdx.x] : 0u;
  uint32_t v[8];
  load8(data, base, n, v);
  block_excl_scan8(v, sm);
#pragma unroll
  for (int m = 0; m < 8; ++m) v[m] += off;
  store8(data, base, n, v);
}
}  // namespace
// In-place exclusive scan of data[0..n); scratch must hold >= n/2048 + n/2048^2 + 8 words.
int grpic_exclusive_scan(uint32_t* data, size_t n, uint32_t* scratch, cudaStream_t st) {
  const size_t nb = (n + kScanTile - 1) / kScanTile;
  if (nb <= 1) {
    scan_tiles_kernel<<<1, kThreads, 0, st>>>(data, n, nullptr);
    grpic_count_launches(1);
    return grpic_launch_ok();
  }
  // reduce - scan the tile sums - scan the tiles with their offsets: the data is read twice and
  // written once (the round-1 form scanned, then added: two reads, two writes, word by word)
  grpic_count_launches(2);
  tile_sums_kernel<<<(unsigned)nb, kThreads, 0, st>>>(data, n, scratch);
  int rc = grpic_exclusive_scan(scratch, nb, scratch + nb, st);
  if (rc != GRPIC_OK) return rc;
  scan_tiles_kernel<<<(unsigned)nb, kThreads, 0, st>>>(data, n, scratch);
  return grpic_launch_ok();
}
namespace {

// ------------------------------------------------------------------ radix sort passes
__device__ __forceinline__ uint32_t make_key(uint32_t cell, uint32_t flag, uint32_t ncells) {
  return (flag & 2u) ? ncells : min(cell, ncells);
}

// per-tile digit histogram -> hist[digit*ntiles + tile].  Every thread takes 8 CONSECUTIVE keys (two
// 16-byte loads), merges runs of equal digit among them (in the last pass, and in the first one of
// an already cell-ordered array, all eight are usually equal) and adds each run once to its warp's
// private histogram in shared memory; thread d then sums the eight warp histograms of digit d.
template <bool FIRST>
__global__ void __launch_bounds__(kThreads)
radix_hist_kernel(const uint32_t* keys, const uint32_t* cell, const uint32_t* flag, int64_t n,
                  uint32_t ncells, int shift, uint32_t* hist, uint32_t ntiles) {
  __shared__ uint32_t sh[kThreads / 32][kRadix];
  const int w = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < kThreads / 32; ++q) sh[q][threadIdx.x] = 0;
  __syncthreads();
  const int64_t e0 = (int64_t)blockIdx.x * kTile + (int64_t)threadIdx.x * 8;
  uint32_t k[8];
  int cnt = 0;
  // the caller's cell / flag arrays are only promised 4-byte alignment: vector loads if they have 16
  const bool vec = !FIRST || ((((uintptr_t)cell | (uintptr_t)flag) & 15u) == 0);
  if (e0 + 8 <= n && vec) {
    cnt = 8;
    if (FIRST) {
      const uint4 c0 = *reinterpret_cast<const uint4*>(cell + e0), c1 = *reinterpret_cast<const uint4*>(cell + e0 + 4);
      const uint4 f0 = *reinterpret_cast<const uint4*>(flag + e0), f1 = *reinterpret_cast<const uint4*>(flag + e0 + 4);
      k[0] = make_key(c0.x, f0.x, ncells); k[1] = make_key(c0.y, f0.y, ncells);
      k[2] = make_key(c0.z, f0.z, ncells); k[3] = make_key(c0.w, f0.w, ncells);
      k[4] = make_key(c1.x, f1.x, ncells); k[5] = make_key(c1.y, f1.y, ncells);
      k[6] = make_key(c1.z, f1.z, ncells); k[7] = make_key(c1.w, f1.w, ncells);
    } else {
      const uint4 a = *reinterpret_cast<const uint4*>(keys + e0), b = *reinterpret_cast<const uint4*>(keys + e0 + 4);
      k[0] = a.x; k[1] = a.y; k[2] = a.z; k[3] = a.w; k[4] = b.x; k[5] = b.y; k[6] = b.z; k[7] = b.w;
    }
  } else {
    for (int m = 0; m < 8; ++m)
      if (e0 + m < n) { k[m] = FIRST ? make_key(cell[e0 + m], flag[e0 + m], ncells) : keys[e0 + m]; cnt = m + 1; }
  }
  uint32_t run_d = 0, run_n = 0;
#pragma unroll
  for (int m = 0; m < 8; ++m) {
    if (m < cnt) {
      const uint32_t d = (k[m] >> shift) & 0xFFu;
      if (run_n && d == run_d) { ++run_n; }
      else {
        if (run_n) atomicAdd(&sh[w][run_d], run_n);
        run_d = d; run_n = 1;
      }
    }
  }
  if (run_n) atomicAdd(&sh[w][run_d], run_n);
  __syncthreads();
  uint32_t tot = 0;
#pragma unroll
  for (int q = 0; q < kThreads / 32; ++q) tot += sh[q][threadIdx.x];
  hist[(size_t)threadIdx.x * ntiles + blockIdx.x] = tot;
}

// stable scatter of one tile: warp w owns keys [w*256, w*256+256) of the tile in 8 groups.
// The tile is first sorted by digit in shared memory (position = exclusive prefix of the tile's digit
// counts + stable rank of the key among the tile's keys of that digit), then written out in that
// order: all keys of one digit go to consecutive global positions, so every warp store covers whole
// runs instead of 32 scattered 4-byte elements (pass 1 at 1e8 keys: 1.08 -> see profiles/r02_final.md).
// resident CTAs per SM asked of the compiler (register cap 64): measured steady-state sort at 1e8
// particles 5.25 / 5.39 / 5.72 ms for 4 / 5 / 6 (5 and 6 spill)
#ifndef GRPIC_SCATTER_MINB
#define GRPIC_SCATTER_MINB 4
#endif
template <bool FIRST>
__global__ void __launch_bounds__(kThreads, GRPIC_SCATTER_MINB)
radix_scatter_kernel(const uint32_t* keys_in, const uint32_t* idx_in, const uint32_t* cell,
                     const uint32_t* flag, int64_t n, uint32_t ncells, int shift,
                     const uint32_t* hist_scanned, uint32_t ntiles, uint32_t* keys_out,
                     uint32_t* idx_out) {
  __shared__ uint32_t whist[kThreads / 32][kRadix];   // per-warp digit counts, then local starts
  __shared__ uint32_t gdelta[kRadix];                  // global start of the tile's run of a digit - its start in the tile
  __shared__ uint32_t skey[kTile], sidx[kTile];
  __shared__ uint32_t wsum[kThreads / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < kThreads / 32; ++q) whist[q][threadIdx.x] = 0;
  __syncthreads();
  const int64_t tbase = (int64_t)blockIdx.x * kTile;
  const int64_t wbase = tbase + (int64_t)w * (kGroups * 32);
  uint32_t key[kGroups], idx[kGroups], dig[kGroups];
  // global start of the tile's run of digit threadIdx.x: asked for now, used in step 2
  const uint32_t gs = hist_scanned[(size_t)threadIdx.x * ntiles + blockIdx.x];
  // all sixteen loads first (written as key = flag & 2 ? ncells : min(cell, ncells) inside the loop,
  // the compiler loads the flag, branches on it and only then loads the cell: sixteen dependent
  // round trips, 1.05 ms for the first pass against 0.57 for the second at 1e8 keys)
#pragma unroll
  for (int q = 0; q < kGroups; ++q) {
    const int64_t e = wbase + q * 32 + lane;
    const int64_t es = e < n ? e : 0;
    key[q] = FIRST ? cell[es] : keys_in[es];
    idx[q] = FIRST ? flag[es] : idx_in[es];
  }
#pragma unroll
  for (int q = 0; q < kGroups; ++q) {
    const int64_t e = wbase + q * 32 + lane;
    if (FIRST) {
      const uint32_t c = min(key[q], ncells);
      key[q] = (idx[q] & 2u) ? ncells : c;
      idx[q] = (uint32_t)e;
    }
    dig[q] = (key[q] >> shift) & 0xFFu;
    if (e >= n) { key[q] = 0; idx[q] = 0; dig[q] = 0x100u; }   // sentinel: never ranked or written
  }
  // 1. per-warp digit counts and, in the same sweep, the rank of every key among the keys of its
  //    digit in its warp (input order: group by group, lane by lane).  One MATCH per key -- the
  //    slowest instruction of the kernel -- and one shared-memory update per distinct digit of a group
  const uint32_t lt = (1u << lane) - 1u;
  uint32_t rank_q[kGroups];
#pragma unroll
  for (int q = 0; q < kGroups; ++q) {
    // (MATCH.ANY executes on the ADU pipe at about one per 6 cycles per SM: 25 M of them are 0.5 ms per
    // pass at 1e8 keys, which is what a pass takes.  Forming the peer mask of some of the eight groups on
    // the ALUs instead -- one ballot per digit bit -- was measured: steady-state sort 5.06 / 5.09 / 5.16 /
    // 5.22 / 5.26 ms for 0 / 2 / 3 / 4 / 5 groups by ballot; profiles/r02_late_experiments.md)
    const uint32_t peers = __match_any_sync(0xffffffffu, dig[q]);
    const bool valid = dig[q] < kRadix;
    const uint32_t before = valid ? whist[w][dig[q]] : 0u;
    __syncwarp();
    if (valid && lane == (__ffs(peers) - 1)) whist[w][dig[q]] = before + __popc(peers);
    __syncwarp();
    rank_q[q] = before + __popc(peers & lt);
  }
  __syncthreads();
  // 2. thread d: tile count of digit d, exclusive prefix over the digits (block scan), local start
  //    of every warp's run inside the tile's sorted order, global start of the tile's run
  {
    uint32_t tot = 0;
#pragma unroll
    for (int q = 0; q < kThreads / 32; ++q) tot += whist[q][threadIdx.x];
    uint32_t incl = tot;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += t;
    }
    if (lane == 31) wsum[w] = incl;
    __syncthreads();
    uint32_t off = 0;
    for (int q = 0; q < w; ++q) off += wsum[q];
    uint32_t run = off + incl - tot;                 // exclusive prefix of digit threadIdx.x
    // element e of the sorted tile, of digit d, goes to global position e + gdelta[d]
    gdelta[threadIdx.x] = gs - run;
#pragma unroll
    for (int q = 0; q < kThreads / 32; ++q) {
      const uint32_t cnt = whist[q][threadIdx.x];
      whist[q][threadIdx.x] = run;
      run += cnt;
    }
  }
  __syncthreads();
  // 3. position in the tile's sorted order = start of the warp's run of the digit + rank in the warp
#pragma unroll
  for (int q = 0; q < kGroups; ++q) {
    if (dig[q] < kRadix) {
      const uint32_t pos = whist[w][dig[q]] + rank_q[q];
      skey[pos] = key[q];
      sidx[pos] = idx[q];
    }
  }
  __syncthreads();
  // 4. write the tile in sorted order
  const uint32_t cnt_tile = (uint32_t)((n - tbase) < (int64_t)kTile ? (n - tbase) : (int64_t)kTile);
#pragma unroll
  for (int m = 0; m < kTile / kThreads; ++m) {
    const uint32_t e = m * kThreads + threadIdx.x;
    if (e < cnt_tile) {
      const uint32_t k = skey[e], d = (k >> shift) & 0xFFu;
      const uint32_t pos = e + gdelta[d];
      keys_out[pos] = k;
      idx_out[pos] = sidx[e];
    }
  }
}

// Payload move by the final permutation.  All nine loads are issued before the first store: the
// arrays carry no no-alias promise, so written as nine copy statements the compiler keeps every
// load behind the previous store (ten dependent memory round trips per thread; 2.88 ms at 1e8
// particles against the time noted in profiles/r02_final.md for this form).  (Loads with the
// L2::64B fetch-size hint were measured: first sort of a random order 23.9 -> 22.9 ms, steady
// state 5.28 -> 5.36 ms; not kept.  Two / four particles per thread, all loads before the first store:
// steady-state sort 5.10 -> 5.11 / 5.15 ms; not kept.)
__global__ void __launch_bounds__(256)
gather_particles_kernel(grpic_particles in, grpic_particles out, const uint32_t* __restrict__ perm,
                        uint32_t* __restrict__ perm_out) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= in.n) return;
  const uint32_t s = perm[k];
  const double x1 = in.x1[s], x2 = in.x2[s], x3 = in.x3[s];
  const double u1 = in.u1[s], u2 = in.u2[s], u3 = in.u3[s];
  const double w = in.w[s];
  const uint32_t cell = in.cell[s], flag = in.flag[s];
  out.x1[k] = x1; out.x2[k] = x2; out.x3[k] = x3;
  out.u1[k] = u1; out.u2[k] = u2; out.u3[k] = u3;
  out.w[k] = w;
  out.cell[k] = cell;
  out.flag[k] = flag;
  if (perm_out) perm_out[k] = s;
}

// ------------------------------------------------------------------ compaction
__global__ void __launch_bounds__(kThreads)
alive_count_kernel(const uint32_t* flag, int64_t n, uint32_t* counts) {
  __shared__ uint32_t sm[kThreads / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t wbase = (int64_t)blockIdx.x * kTile + (int64_t)w * (kGroups * 32);
  uint32_t c = 0;
#pragma unroll
  for (int q = 0; q < kGroups; ++q) {
    const int64_t e = wbase + q * 32 + lane;
    const bool alive = (e < n) && !(flag[e] & 2u);
    c += __popc(__ballot_sync(0xffffffffu, alive));
  }
  if (lane == 0) sm[w] = c;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = 0;
    for (int q = 0; q < kThreads / 32; ++q) t += sm[q];
    counts[blockIdx.x] = t;
  }
}

__global__ void __launch_bounds__(kThreads)
compact_scatter_kernel(grpic_particles in, grpic_particles out, const uint32_t* offsets,
                       uint32_t ntiles, int64_t* n_alive) {
  __shared__ uint32_t sm[kThreads / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t wbase = (int64_t)blockIdx.x * kTile + (int64_t)w * (kGroups * 32);
  uint32_t ballots[kGroups];
  uint32_t c = 0;
#pragma unroll
  for (int q = 0; q < kGroups; ++q) {
    const int64_t e = wbase + q * 32 + lane;
    const bool alive = (e < in.n) && !(in.flag[e] & 2u);
    ballots[q] = __ballot_sync(0xffffffffu, alive);
    c += __popc(ballots[q]);
  }
  if (lane == 0) sm[w] = c;
  __syncthreads();
  uint32_t off = offsets[blockIdx.x];
  uint32_t tile_total = 0;
  for (int q = 0; q < kThreads / 32; ++q) {
    if (q < w) off += sm[q];
    tile_total += sm[q];
  }
  if (blockIdx.x == ntiles - 1 && threadIdx.x == 0)
    *n_alive = (int64_t)offsets[blockIdx.x] + (int64_t)tile_total;
  const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
  for (int q = 0; q < kGroups; ++q) {
    const int64_t e = wbase + q * 32 + lane;
    if (ballots[q] & (1u << lane)) {
      const uint32_t d = off + __popc(ballots[q] & lt);
      const double x1 = in.x1[e], x2 = in.x2[e], x3 = in.x3[e];      // loads before stores (see
      const double u1 = in.u1[e], u2 = in.u2[e], u3 = in.u3[e];      // gather_particles_kernel)
      const double w8 = in.w[e];
      const uint32_t cell = in.cell[e], flag = in.flag[e];
      out.x1[d] = x1; out.x2[d] = x2; out.x3[d] = x3;
      out.u1[d] = u1; out.u2[d] = u2; out.u3[d] = u3;
      out.w[d] = w8;
      out.cell[d] = cell;
      out.flag[d] = flag;
    }
    off += __popc(ballots[q]);
  }
}
// entries [n_alive, n) of the output are marked removed, so the caller may keep using n as an
// upper bound without reading n_alive back.
__global__ void mark_tail_kernel(grpic_particles out, int64_t n, const int64_t* n_alive) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n && k >= *n_alive) {
    out.flag[k] = 2u;
    out.cell[k] = 0xFFFFFFFFu;
  }
}

bool ptc_ok(const grpic_particles* p) {
  return p && p->n >= 0 &&
         (p->n == 0 || (p->x1 && p->x2 && p->x3 && p->u1 && p->u2 && p->u3 && p->w && p->cell && p->flag));
}


// ------------------------------------------------------------------ contention-free cell order
// start[c] = first position of key c in the sorted key array (lower bound), c in [0, ncells + 1]:
// start[ncells] = first removed particle, start[ncells + 1] = n.
// One thread per four sorted keys: wherever the key steps up from a to b at position k, start[c] = k
// for every c in (a, b]; position n closes the list with the sentinel ncells + 1.  (Streams the keys
// once; the round-1 form was a binary search per cell: 27 dependent loads, 132 us at 1e8 keys.)
__global__ void __launch_bounds__(256)
cell_start_kernel(const uint32_t* __restrict__ keys, uint32_t n, uint32_t ncells, uint32_t* __restrict__ start) {
  const uint64_t k0 = 4ull * ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x);
  if (k0 > n) return;
  uint32_t kv[4];
  if (k0 + 4 <= n && (((uintptr_t)keys) & 15u) == 0) {
    const uint4 a = *reinterpret_cast<const uint4*>(keys + k0);
    kv[0] = a.x; kv[1] = a.y; kv[2] = a.z; kv[3] = a.w;
  } else {
#pragma unroll
    for (int m = 0; m < 4; ++m) kv[m] = (k0 + m < n) ? keys[k0 + m] : ncells + 1u;
  }
  uint32_t lo = k0 == 0 ? 0u : keys[k0 - 1] + 1u;      // first cell whose start is not yet known
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    if (k0 + m <= n) {
      for (uint32_t c = lo; c <= kv[m]; ++c) start[c] = (uint32_t)(k0 + m);
      lo = kv[m] + 1u;
    }
  }
}
// Inside every block of B consecutive cells the particles are re-ordered rank-major: first the
// first particle of each cell, then the second of each, ...  (rank = position among the particles
// of the same cell in the stable order).  Consecutive lanes of the push then sit in DIFFERENT,
// adjacent cells: their 24 gather loads and 8-21 REDs fall into few sectors but never on one
// address (same-address lanes of a RED serialise in L2: 7.0 ms for the plainly sorted order against
// 5.55 ms for this one at 1e8 particles, profiles/r02f).  One warp owns 32 consecutive cells
// (32 / B blocks), lane = cell; perm2[dest] = perm[start[cell] + rank].
__global__ void __launch_bounds__(256)
interleave_perm_kernel(const uint32_t* __restrict__ perm, const uint32_t* __restrict__ start, uint32_t n,
                       uint32_t ncells, uint32_t B, uint32_t* __restrict__ perm2) {
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t cell = (blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32u + lane;
  const uint32_t s = cell < ncells ? start[cell] : 0u;
  const uint32_t cnt = cell < ncells ? start[cell + 1] - s : 0u;
  const uint32_t g0 = lane & ~(B - 1u);                       // first lane of this lane's block
  const uint32_t gmask = (B == 32u ? 0xffffffffu : ((1u << B) - 1u)) << g0;
  uint32_t dest = __shfl_sync(0xffffffffu, s, g0);            // block start (cells are contiguous in the sorted array)
  uint32_t maxc = cnt;
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) maxc = max(maxc, __shfl_xor_sync(0xffffffffu, maxc, d));
  const uint32_t lt = (1u << lane) - 1u;
  for (uint32_t r0 = 0; r0 < maxc; r0 += 4) {               // four ranks per trip: four loads in flight
    uint32_t v[4];
#pragma unroll
    for (uint32_t m = 0; m < 4; ++m) v[m] = (cnt > r0 + m) ? perm[s + r0 + m] : 0u;
#pragma unroll
    for (uint32_t m = 0; m < 4; ++m) {
      const bool act = cnt > r0 + m;
      const uint32_t gb = __ballot_sync(0xffffffffu, act) & gmask;
      if (act) perm2[dest + __popc(gb & lt)] = v[m];
      dest += __popc(gb);
    }
  }
  // removed particles keep their stable order at the tail
  const uint32_t t0 = start[ncells];
  for (uint32_t k = t0 + blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) perm2[k] = perm[k];
}

// stable LSD radix sort of (key, index), then the payload gather; interleave = 0: plain stable
// order, else the rank-major order inside blocks of `interleave` cells
int sort_impl(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out, uint32_t* perm, int interleave,
              cudaStream_t st) {
  if (!ctx || !ptc_ok(in) || !out) return GRPIC_ERR_ARG;
  const int64_t n = in->n;
  out->n = n;
  if (n == 0) return GRPIC_OK;
  if (!ptc_ok(out) || out->x1 == in->x1 || n > 0xFFFFFFF0LL) return GRPIC_ERR_ARG;
  const size_t nA = ((size_t)n + 63) & ~(size_t)63;
  const uint32_t ntiles = (uint32_t)((n + kTile - 1) / kTile);
  const size_t nh = (size_t)kRadix * ntiles;
  const uint32_t ncells = (uint32_t)ctx->g.nr * (uint32_t)ctx->g.nth;
  const size_t nstart = interleave ? (((size_t)ncells + 2 + 63) & ~(size_t)63) : 0;
  const size_t need = (4 * nA + nh + nh / kScanTile + 4096 + nstart) * sizeof(uint32_t);
  if (!ctx->ws || ctx->ws_bytes < need) return GRPIC_ERR_WORKSPACE;
  uint32_t* kA = (uint32_t*)ctx->ws;
  uint32_t* kB = kA + nA;
  uint32_t* iA = kB + nA;
  uint32_t* iB = iA + nA;
  uint32_t* hist = iB + nA;
  uint32_t* scratch = hist + nh;
  uint32_t* start = scratch + nh / kScanTile + 4096;
  int bits = 0;
  while ((1ull << bits) <= (unsigned long long)ncells) ++bits;   // keys in [0, ncells]
  const int passes = (bits + 7) / 8;
  uint32_t *kin = kA, *kout = kB, *iin = iA, *iout = iB;
  for (int p = 0; p < passes; ++p) {
    const int shift = 8 * p;
    if (p == 0) {
      radix_hist_kernel<true><<<ntiles, kThreads, 0, st>>>(nullptr, in->cell, in->flag, n, ncells, shift, hist, ntiles);
    } else {
      radix_hist_kernel<false><<<ntiles, kThreads, 0, st>>>(kin, nullptr, nullptr, n, ncells, shift, hist, ntiles);
    }
    int rc = grpic_exclusive_scan(hist, nh, scratch, st);
    if (rc != GRPIC_OK) return rc;
    if (p == 0) {
      radix_scatter_kernel<true><<<ntiles, kThreads, 0, st>>>(nullptr, nullptr, in->cell, in->flag, n, ncells,
                                                              shift, hist, ntiles, kout, iout);
    } else {
      radix_scatter_kernel<false><<<ntiles, kThreads, 0, st>>>(kin, iin, nullptr, nullptr, n, ncells, shift,
                                                               hist, ntiles, kout, iout);
    }
    uint32_t* t = kin; kin = kout; kout = t;
    t = iin; iin = iout; iout = t;
    grpic_count_launches(2);
  }
  if (interleave) {
    // (moving the payload inside the rank loop instead of writing perm2 first was measured: 24.7 ms
    // against 6.7 ms -- the loop is latency-bound, the separate gather runs at 4.6 TB/s)
    cell_start_kernel<<<(unsigned)(((uint64_t)n / 4 + 1 + 255) / 256), 256, 0, st>>>(kin, (uint32_t)n, ncells, start);
    interleave_perm_kernel<<<(ncells + 255) / 256, 256, 0, st>>>(iin, start, (uint32_t)n, ncells, (uint32_t)interleave, iout);
    uint32_t* t = iin; iin = iout; iout = t;
    grpic_count_launches(2);
  }
  grpic_count_launches(1);
  gather_particles_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(*in, *out, iin, perm);
  return grpic_launch_ok();
}
}  // namespace

extern "C" {

int grpic_sort(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out, uint32_t* perm, void* stream) {
  return sort_impl(ctx, in, out, perm, 0, (cudaStream_t)stream);
}

int grpic_sort_interleaved(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out, uint32_t* perm,
                           int32_t block_cells, void* stream) {
  if (block_cells < 1 || block_cells > 32 || (block_cells & (block_cells - 1))) return GRPIC_ERR_ARG;
  return sort_impl(ctx, in, out, perm, block_cells, (cudaStream_t)stream);
}

// Device address of g_compact_static_scratch on the CURRENT device, resolved once per device (no
// allocation: the array is part of the loaded module) and cached.
static int static_scratch(uint32_t** out) {
  constexpr int kMaxDevices = 64;
  static uint32_t* cache[kMaxDevices] = {};
  static std::mutex mu;
  int dev = -1;
  GRPIC_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return GRPIC_ERR_CUDA;
  std::lock_guard<std::mutex> lock(mu);
  if (!cache[dev]) {
    uint32_t* ptr = nullptr;
    GRPIC_CUDA_OK(cudaGetSymbolAddress((void**)&ptr, g_compact_static_scratch));
    if (!ptr) return GRPIC_ERR_CUDA;
    cache[dev] = ptr;
  }
  *out = cache[dev];
  return GRPIC_OK;
}

int grpic_compact_static(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out, int64_t* n_alive,
                         void* stream) {
  if (!ctx || !ptc_ok(in) || !out || !n_alive) return GRPIC_ERR_ARG;
  const int64_t n = in->n;
  if (n > (int64_t)GRPIC_COMPACT_STATIC_MAX_PARTICLES) return GRPIC_ERR_TOO_LARGE;
  out->n = n;
  cudaStream_t st = (cudaStream_t)stream;
  if (n == 0) {
    GRPIC_CUDA_OK(cudaMemsetAsync(n_alive, 0, sizeof(int64_t), st));
    return GRPIC_OK;
  }
  if (!ptc_ok(out) || out->x1 == in->x1) return GRPIC_ERR_ARG;
  const uint32_t ntiles = (uint32_t)((n + kTile - 1) / kTile);
  static_assert((GRPIC_COMPACT_STATIC_MAX_PARTICLES + kTile - 1) / kTile +
                        (GRPIC_COMPACT_STATIC_MAX_PARTICLES + kTile - 1) / kTile / kScanTile + 4096 <=
                    kStaticScratchWords,
                "static scratch too small for GRPIC_COMPACT_STATIC_MAX_PARTICLES");
  uint32_t* counts = nullptr;
  int rc = static_scratch(&counts);
  if (rc != GRPIC_OK) return rc;
  // nothing in the scratch has to start at zero: alive_count writes counts[0, ntiles), the scan writes
  // every tile sum before it reads it -- the previous call's contents are never read
  uint32_t* scratch = counts + ntiles;
  alive_count_kernel<<<ntiles, kThreads, 0, st>>>(in->flag, n, counts);
  rc = grpic_exclusive_scan(counts, ntiles, scratch, st);
  if (rc != GRPIC_OK) return rc;
  compact_scatter_kernel<<<ntiles, kThreads, 0, st>>>(*in, *out, counts, ntiles, n_alive);
  mark_tail_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(*out, n, n_alive);
  grpic_count_launches(3);
  return grpic_launch_ok();
}

int grpic_compact(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out, int64_t* n_alive, void* stream) {
  if (!ctx || !ptc_ok(in) || !out || !n_alive) return GRPIC_ERR_ARG;
  const int64_t n = in->n;
  out->n = n;
  cudaStream_t st = (cudaStream_t)stream;
  if (n == 0) {
    GRPIC_CUDA_OK(cudaMemsetAsync(n_alive, 0, sizeof(int64_t), st));
    return GRPIC_OK;
  }
  if (!ptc_ok(out) || out->x1 == in->x1 || n > 0xFFFFFFF0LL) return GRPIC_ERR_ARG;
  const uint32_t ntiles = (uint32_t)((n + kTile - 1) / kTile);
  const size_t need = ((size_t)ntiles + ntiles / kScanTile + 4096) * sizeof(uint32_t);
  if (!ctx->ws || ctx->ws_bytes < need) return GRPIC_ERR_WORKSPACE;
  uint32_t* counts = (uint32_t*)ctx->ws;
  uint32_t* scratch = counts + ntiles;
  alive_count_kernel<<<ntiles, kThreads, 0, st>>>(in->flag, n, counts);
  int rc = grpic_exclusive_scan(counts, ntiles, scratch, st);
  if (rc != GRPIC_OK) return rc;
  compact_scatter_kernel<<<ntiles, kThreads, 0, st>>>(*in, *out, counts, ntiles, n_alive);
  mark_tail_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(*out, n, n_alive);
  grpic_count_launches(3);
  return grpic_launch_ok();
}

}  // extern "C"
