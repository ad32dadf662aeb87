// scan_dup.cu — A5/A6/A7b/A8 for sm_100a: compaction scan (+ depth digit counts) with the tile-grid prefix (ranges, D) as a
// role of its first CTA, and the row scatter that writes the per-tile lists in depth order without sorting the pairs.
#include "common.cuh"

namespace fdgs {

// ---------------------------------------------------------------------------------------------
// Single-pass chained scan with decoupled look-back.  state word: flag << 62 | value,
// flag 1 = tile aggregate, 2 = inclusive prefix.  Tiles take dynamic ids from a ticket so that every
// predecessor of a waiting tile is already running.
constexpr unsigned long long FLAG_AGG = 1ull << 62, FLAG_PRE = 2ull << 62, VAL_MASK = (1ull << 62) - 1;

__device__ __forceinline__ unsigned int block_exclusive_scan(unsigned int v, unsigned int& total, unsigned int* warp_sums) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned int incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const unsigned int n = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += n; }
  if (lane == 31) warp_sums[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    unsigned int w = lane < (int)(blockDim.x >> 5) ? warp_sums[lane] : 0, wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned int n = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += n; }
    warp_sums[lane] = wi - w;
    if (lane == 31) warp_sums[32] = wi;
  }
  __syncthreads();
  total = warp_sums[32];
  const unsigned int res = warp_sums[warp] + incl - v;
  __syncthreads();
  return res;
}

// exclusive prefix of all earlier tiles (called by the whole block; warp 0 walks back 32 tiles at a time)
__device__ __forceinline__ unsigned int lookback_prefix(volatile unsigned long long* state, const unsigned int tile,
                                                        const unsigned int aggregate, unsigned int* s_bcast) {
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x;
    if (lane == 0) state[tile] = (tile == 0 ? FLAG_PRE : FLAG_AGG) | aggregate;
    unsigned int prefix = 0;
    long long j = (long long)tile - 1 - lane;
    if (tile > 0) {
      while (true) {
        unsigned long long s = FLAG_PRE;   // lanes past the start read as "prefix 0"
        if (j >= 0) { do { s = state[j]; } while ((s >> 62) == 0); }
        const unsigned int pre_mask = __ballot_sync(0xffffffffu, (s >> 62) == 2);
        const int first = pre_mask ? __ffs(pre_mask) - 1 : 32;
        unsigned int v = lane <= first ? (unsigned int)(s & VAL_MASK) : 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        prefix += v;
        if (pre_mask) break;
        j -= 32;
      }
      if (lane == 0) state[tile] = FLAG_PRE | (unsigned long long)(prefix + aggregate);
    }
    if (lane == 0) *s_bcast = prefix;
  }
  __syncthreads();
  return *s_bcast;
}

// Tile grid (role of CTA 0 of the compaction launch): 2D inclusive prefix of the coverage difference array = list length
// of every tile; its exclusive scan in tile order = the tile ranges (A8) and D.  One CTA, all in shared memory:
// rows by warps (shuffle scans), columns by threads, then a blocked scan over the tiles.
__device__ void tile_grid_role(const int* __restrict__ tile_diff, const int tiles_x, const int tiles_y, const unsigned int cap,
                               WsHeader* hdr, const WsHeader mirror, uint2* __restrict__ ranges, int* grid, unsigned int* warp_sums) {
  const int sx = tiles_x + 1, rows = tiles_y + 1, cells = sx * rows, tiles = tiles_x * tiles_y;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  for (int i0 = threadIdx.x; i0 < cells; i0 += 8 * blockDim.x) {      // eight independent loads per thread in flight
    int v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = i0 + k * (int)blockDim.x < cells ? tile_diff[i0 + k * blockDim.x] : 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) if (i0 + k * (int)blockDim.x < cells) grid[i0 + k * blockDim.x] = v[k];
  }
  __syncthreads();
  for (int y = warp; y < rows; y += nwarps) {             // inclusive scan along x, one warp per row
    int carry = 0;
    for (int x0 = 0; x0 < sx; x0 += 32) {
      const int x = x0 + lane;
      int v = x < sx ? grid[y * sx + x] : 0;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int n = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += n; }
      v += carry;
      if (x < sx) grid[y * sx + x] = v;
      carry = __shfl_sync(0xffffffffu, v, 31);
    }
  }
  __syncthreads();
  // columns by threads; eight loads in flight per step (a load never aliases the stores of the same step: another row)
  for (int x = threadIdx.x; x < sx; x += blockDim.x) {
    int run = 0;
    for (int y0 = 0; y0 < rows; y0 += 8) {
      int v[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) v[k] = y0 + k < rows ? grid[(y0 + k) * sx + x] : 0;
#pragma unroll
      for (int k = 0; k < 8; ++k) { run += v[k]; if (y0 + k < rows) grid[(y0 + k) * sx + x] = run; }
    }
  }
  __syncthreads();
  // exclusive scan over tiles in row-major order; each thread owns a contiguous chunk and walks it as (row, column)
  const int per = (tiles + blockDim.x - 1) / blockDim.x, t0 = min((int)threadIdx.x * per, tiles), t1 = min(t0 + per, tiles);
  const int ty0 = t0 / tiles_x, tx0 = t0 - ty0 * tiles_x;
  unsigned int sum = 0;
  for (int t = t0, ty = ty0, tx = tx0; t < t1; ++t) {
    sum += (unsigned int)grid[ty * sx + tx];
    if (++tx == tiles_x) { tx = 0; ++ty; }
  }
  unsigned int total;
  unsigned int run = block_exclusive_scan(sum, total, warp_sums);
  const bool overflow = total > cap;
  for (int t = t0, ty = ty0, tx = tx0; t < t1; ++t) {
    const unsigned int c = (unsigned int)grid[ty * sx + tx];
    ranges[t] = overflow ? make_uint2(0, 0) : make_uint2(run, run + c);
    run += c;
    if (++tx == tiles_x) { tx = 0; ++ty; }
  }
  if (threadIdx.x == 0) {
    hdr->num_pairs = overflow ? 0u : total; hdr->overflow = overflow ? 1u : 0u; hdr->total_pairs = total;
    hdr->N = mirror.N; hdr->K = mirror.K; hdr->W = mirror.W; hdr->H = mirror.H; hdr->pair_capacity = mirror.pair_capacity; hdr->tiles = mirror.tiles;
  }
}

// Compaction: survivors (tiles_touched > 0) in primitive-id order -> (depth bits, id) pairs, plus the digit counts of
// the four 8-bit passes of the depth sort (the keys are in registers here: the sort never reads them just to count).
// CTA 0 of the launch does not compact: it runs the tile-grid role above, which depends on the preprocess kernel only
// and would otherwise be a one-CTA launch of its own on the critical path.
__global__ void __launch_bounds__(SCAN_THREADS) compact_kernel(const unsigned int* __restrict__ tiles_touched,
                                                               const SplatRec* __restrict__ rec, const int N, WsHeader* hdr,
                                                               unsigned long long* state, unsigned int* __restrict__ keys,
                                                               unsigned int* __restrict__ vals, unsigned int* __restrict__ vis_ids,
                                                               unsigned int* __restrict__ sort_hist, const int* __restrict__ tile_diff,
                                                               const int tiles_x, const int tiles_y, const unsigned int cap,
                                                               const WsHeader mirror, uint2* __restrict__ ranges, const unsigned int key_base) {
  extern __shared__ int grid[];                 // (tiles_y+1) x (tiles_x+1), used by CTA 0 only
  __shared__ unsigned int warp_sums[33], s_tile, s_prefix, hist[4][RADIX];
  if (blockIdx.x == 0) {
    tile_grid_role(tile_diff, tiles_x, tiles_y, cap, hdr, mirror, ranges, grid, warp_sums);
    return;
  }
  if (threadIdx.x == 0) s_tile = atomicAdd(&hdr->scan_ticket[0], 1u);
#pragma unroll
  for (int p = 0; p < 4; ++p) { hist[p][threadIdx.x] = 0; hist[p][threadIdx.x + SCAN_THREADS] = 0; }     // RADIX == 2 SCAN_THREADS
  __syncthreads();
  const unsigned int tile = s_tile;
  const long long base = (long long)tile * SCAN_TILE + (long long)threadIdx.x * SCAN_ITEMS;
  unsigned int flags = 0, cnt = 0;   // SCAN_ITEMS <= 32 bits
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k)
    if (base + k < N && tiles_touched[base + k] > 0) { flags |= 1u << k; ++cnt; }
  unsigned int total;
  const unsigned int excl = block_exclusive_scan(cnt, total, warp_sums);
  const unsigned int prefix = lookback_prefix(state, tile, total, &s_prefix);
  unsigned int pos = prefix + excl;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k)
    if (flags & (1u << k)) {
      const unsigned int key = __float_as_uint(rec[base + k].depth) - key_base;      // z > znear: the difference keeps the order of the bits
      keys[pos] = key; vals[pos] = (unsigned int)(base + k); vis_ids[pos] = (unsigned int)(base + k); ++pos;
      // digit counts of the four depth passes.  The two low digits of an fp32 depth are spread over all 512 bins; the two
      // high ones (exponent and top mantissa bits) take a handful of values in a whole scene, so a plain shared atomic would
      // serialise the CTA on one or two addresses (38 % of this kernel's stall samples): the lanes that are here together
      // are grouped by digit first and one of each group adds the group's size
      atomicAdd(&hist[0][key & (RADIX - 1)], 1u);
      atomicAdd(&hist[1][(key >> RADIX_BITS) & (RADIX - 1)], 1u);
      const unsigned int am = __activemask();
#pragma unroll
      for (int p = 2; p < 4; ++p) {
        const unsigned int d = (key >> (RADIX_BITS * p)) & (RADIX - 1);
        const unsigned int peers = __match_any_sync(am, d);
        if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&hist[p][d], (unsigned int)__popc(peers));
      }
    }
  if (tile == gridDim.x - 2 && threadIdx.x == 0) hdr->num_visible = prefix + total;    // gridDim.x - 1 compaction tiles
  __syncthreads();
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int h = 0; h < RADIX / SCAN_THREADS; ++h) {
      const unsigned int v = hist[p][threadIdx.x + h * SCAN_THREADS];
      if (v) atomicAdd(sort_hist + p * RADIX + threadIdx.x + h * SCAN_THREADS, v);
    }
}

// ---------------------------------------------------------------------------------------------
// A6/A7, level 2: the per-tile lists in depth order, written straight to their final place ("row scatter").
//
// Survivors arrive sorted by depth (level 1) together with their tile rectangles (ys = y0 | y1 << 16, xs = x0 | x1 << 16,
// gathered by the last pass of the depth sort).  The list of tile T is {j : T in rect[j]} in ascending j, stored at
// [ranges[T].x, ranges[T].y): a stable partition of the emission order by tile — what a stable sort of the (tile, id)
// pairs by tile id produces.  The ranges are already known from the coverage grid, and the covered sets are rectangles,
// i.e. x-intervals in every tile row, so no sort is needed.  One CTA owns (chunk c of RS-chunk consecutive survivors,
// tile row y, block of RS_XB tile columns):
//   1. filter: which survivors of the chunk cover the row is read from the ballot words of row_ballot_kernel (one word
//      per 32 survivors, computed once for all rows); the hits stay in depth order; their x-intervals go into a 1D
//      difference array, whose prefix is the chunk's count for every tile of the row;
//   2. the counts are published at once and the exclusive prefix over the earlier chunks of the same row is fetched by
//      decoupled look-back (per tile column; chunk ids come from a ticket, so every predecessor is already running);
//      ranges[T].x + that prefix = where this chunk starts writing in tile T;
//   3. ranks inside the chunk: hit h (depth order) sets bit h in the bit mask of every tile it covers; the rank of a
//      hit in a tile is the popcount of the lower bits — a prefix over the mask words plus one masked popcount.  Every
//      (hit, tile) pair then stores its primitive id at its final position.  O(1) work per pair, 4 bytes written per
//      pair; no key array, no sort, no per-pair search.
// Replaces offsets scan + pair emission + 2-pass radix sort of the D pairs (round 1: 146 us per view at cfg3) and the
// first round-2 design (per-chunk 2D coverage tables + ordered scatter in groups of 32 survivors: 150 us — its groups were
// too small to amortise their barriers where the splats are small).
constexpr int RS_THREADS = 256, RS_LC = 512, RS_WORDS = RS_LC / 32, RS_XB = 128;
constexpr unsigned int RS_AGG = 1u << 30, RS_PRE = 2u << 30, RS_MASK = (1u << 30) - 1;

// Row filter of the row scatter, once for all rows: a warp takes 32 consecutive survivors (depth order), loads their row
// ranges once and votes row by row; lane y % 32 keeps the ballot of row y and stores it at (row, iteration).  The scatter
// items (chunk, row) then read their ballots — one word per 32 survivors — instead of every item scanning the whole
// chunk: rows x survivors tests (a third of the scatter's instructions at cfg3, most of them at 8 M Gaussians) become
// survivors / 32 loads plus ~3 instructions per (row, 32 survivors).
__global__ void __launch_bounds__(256) row_ballot_kernel(const WsHeader* __restrict__ hdr, const unsigned int* __restrict__ ys, const int tiles_y,
                                                         const size_t stride, unsigned int* __restrict__ bal) {
  const unsigned int n = hdr->num_visible;
  if (hdr->overflow) return;
  const unsigned int iters = (n + 31) / 32, lane = threadIdx.x & 31;
  const unsigned int gw = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), nw = gridDim.x * (blockDim.x >> 5);
  for (unsigned int it = gw; it < iters; it += nw) {
    const unsigned int j = it * 32 + lane;
    const unsigned int yv = j < n ? ys[j] : 0u;                          // y0 = y1 = 0: covers no row
    const int y0 = (int)(yv & 0xffffu), y1 = (int)(yv >> 16);
    for (int yb = 0; yb < tiles_y; yb += 32) {
      unsigned int mine = 0;
#pragma unroll
      for (int k = 0; k < 32; ++k) {
        const unsigned int b = __ballot_sync(0xffffffffu, y0 <= yb + k && y1 > yb + k);
        if ((int)lane == k) mine = b;
      }
      if (yb + (int)lane < tiles_y) bal[(size_t)(yb + lane) * stride + it] = mine;
    }
  }
}

// 6 CTAs per SM (40 registers): alone the kernel is 4 % faster at the 8 CTAs per SM the compiler picks by itself (32 registers),
// but it never runs alone in a step or in playback — with 6 the other views' front ends find room next to it: step
// 4.503 -> 4.475 ms, four frames in flight 2268 -> 2372 FPS, single frame 0.490 -> 0.493 ms (profiles/r2_front_end_history.md)
__global__ void __launch_bounds__(RS_THREADS, 6) row_scatter_kernel(WsHeader* hdr, const unsigned int* __restrict__ bal, const size_t bal_stride, const unsigned int* __restrict__ xs,
                                                                 const unsigned int* __restrict__ ids, const uint2* __restrict__ ranges,
                                                                 volatile unsigned int* lb_state, const int tiles_x, const int tiles_y,
                                                                 const int xblocks, const unsigned int chunk, unsigned int* __restrict__ pair_ids) {
  __shared__ unsigned int mask[RS_WORDS][RS_XB], pref[RS_WORDS][RS_XB];
  __shared__ unsigned int list_j[RS_LC], list_x[RS_LC];
  __shared__ unsigned int bal_s[RS_MAX_ITERS];
  __shared__ unsigned short off[RS_MAX_ITERS + 2];     // exclusive prefix of the hit counts: <= RS_MAX_CHUNK = 32768
  __shared__ int diff[RS_XB + 1];
  __shared__ unsigned int cursor[RS_XB], s_ticket;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned int n = hdr->num_visible;
  if (hdr->overflow) return;
  const unsigned int per_chunk = (unsigned int)tiles_y * xblocks;
  const int tiles = tiles_x * tiles_y;
  // persistent CTAs: work items (chunk, row, column block) are taken from a ticket, chunk-major, until the survivors run out
  while (true) {
    __syncthreads();                                    // previous item finished with the shared arrays
    if (threadIdx.x == 0) s_ticket = atomicAdd(&hdr->scan_ticket[1], 1u);
    for (int i = threadIdx.x; i <= RS_XB; i += RS_THREADS) diff[i] = 0;
    for (int i = threadIdx.x; i < RS_WORDS * RS_XB; i += RS_THREADS) (&mask[0][0])[i] = 0;
    __syncthreads();
    const unsigned int c = s_ticket / per_chunk, rr = s_ticket % per_chunk;
    if ((unsigned long long)c * chunk >= n) return;     // tickets are dense: every chunk below this one exists
    const int y = rr / xblocks, xbase = (rr % xblocks) * RS_XB, nx = min(RS_XB, tiles_x - xbase);
    const unsigned int j0 = c * chunk, j1 = min(n, j0 + chunk);
    const unsigned int iters = (j1 - j0 + 31) / 32;
    // ---- 1. the survivors of the chunk that cover this row: ballot words of row_ballot_kernel, one per 32 survivors
    //         (survivor j0 + 32 it + i is bit i of word it).  With several column blocks the hits of the other blocks stay
    //         in the list with an empty x-interval. ----
    for (unsigned int it = threadIdx.x; it < iters; it += RS_THREADS) {
      const unsigned int b = bal[(size_t)y * bal_stride + (j0 >> 5) + it];
      bal_s[it] = b; off[it] = (unsigned short)__popc(b);
    }
    __syncthreads();
    if (warp == 0) {                          // exclusive prefix of the per-iteration hit counts
      unsigned int carry = 0;
      for (unsigned int i0 = 0; i0 < iters; i0 += 32) {
        const unsigned int v = i0 + lane < iters ? off[i0 + lane] : 0;
        unsigned int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
        if (i0 + lane < iters) off[i0 + lane] = (unsigned short)(carry + incl - v);
        carry += __shfl_sync(0xffffffffu, incl, 31);
      }
      if (lane == 0) off[iters] = (unsigned short)carry;
    }
    __syncthreads();
    const unsigned int H = off[iters];
    // ---- 2. rounds of up to RS_LC hits (depth order).  The first round also covers the difference array of ALL hits,
    //         the publication of the counts and the look-back. ----
    for (unsigned int r0 = 0; r0 < H || r0 == 0; r0 += RS_LC) {
      if (r0 > 0) {
        __syncthreads();                                // previous round consumed
        for (int i = threadIdx.x; i < RS_WORDS * RS_XB; i += RS_THREADS) (&mask[0][0])[i] = 0;
        __syncthreads();
      }
      // 2a. the hit list of the round, dense: thread it expands the ballot of iteration it
      for (unsigned int it = threadIdx.x; it < iters; it += RS_THREADS) {
        unsigned int bal = bal_s[it], h = off[it];
        while (bal) {
          const int bit = __ffs(bal) - 1;
          bal &= bal - 1;
          if (h >= r0 && h < r0 + RS_LC) list_j[h - r0] = j0 + it * 32 + bit;
          ++h;
        }
      }
      __syncthreads();
      // 2b. one thread per hit: x-interval, bits into the masks of the tiles it covers (first round: every hit of the chunk
      //     also enters the difference array, in strides of RS_LC)
      const unsigned int m = H > r0 ? min((unsigned int)RS_LC, H - r0) : 0u;
      for (unsigned int hl = threadIdx.x; hl < m; hl += RS_THREADS) {
        const unsigned int xw = xs[list_j[hl]];
        const int xa = min(max((int)(xw & 0xffffu) - xbase, 0), nx);           // clamped to the column block; a hit that lies in another
        const unsigned int x0 = (unsigned int)xa, x1 = (unsigned int)max(min((int)(xw >> 16) - xbase, nx), xa);   // block keeps an empty interval
        list_x[hl] = x0 | (x1 << 16);
        if (r0 == 0) { atomicAdd(&diff[x0], 1); atomicAdd(&diff[x1], -1); }
        const unsigned int bitv = 1u << (hl & 31);
        for (unsigned int x = x0; x < x1; ++x) atomicOr(&mask[hl >> 5][x], bitv);
      }
      if (r0 == 0) {
        if (H > RS_LC) {                      // rare: hits beyond the first round still count; walk the ballots for them
          for (unsigned int it = threadIdx.x; it < iters; it += RS_THREADS) {
            unsigned int bal = bal_s[it], h = off[it];
            while (bal) {
              const int bit = __ffs(bal) - 1;
              bal &= bal - 1;
              if (h >= RS_LC) {
                const unsigned int xw = xs[j0 + it * 32 + bit];
                const int xa = min(max((int)(xw & 0xffffu) - xbase, 0), nx);
                atomicAdd(&diff[xa], 1); atomicAdd(&diff[max(min((int)(xw >> 16) - xbase, nx), xa)], -1);
              }
              ++h;
            }
          }
        }
        __syncthreads();
        if (warp == 1) {                      // count of every tile column of the row = prefix of the difference array (RS_XB = 4 x 32)
          int v[4], sum = 0;
#pragma unroll
          for (int k = 0; k < 4; ++k) { sum += diff[lane * 4 + k]; v[k] = sum; }
          int incl = sum;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
#pragma unroll
          for (int k = 0; k < 4; ++k) diff[lane * 4 + k] = incl - sum + v[k];
        }
        __syncthreads();
        // publish the counts, look back over the earlier chunks of this row
        if ((int)threadIdx.x < nx) {
          const int t = y * tiles_x + xbase + threadIdx.x;
          const unsigned int my_count = (unsigned int)diff[threadIdx.x];
          volatile unsigned int* st = lb_state + t;
          st[(size_t)c * tiles] = (c == 0 ? RS_PRE : RS_AGG) | my_count;
          unsigned int excl = 0;
          if (c > 0) {
            for (long long cc = (long long)c - 1; cc >= 0; --cc) {
              unsigned int v;
              while (((v = st[(size_t)cc * tiles]) >> 30) == 0) __nanosleep(64);
              excl += v & RS_MASK;
              if ((v >> 30) == 2) break;
            }
            st[(size_t)c * tiles] = RS_PRE | (excl + my_count);
          }
          cursor[threadIdx.x] = ranges[t].x + excl;
        }
      }
      __syncthreads();                                  // masks and list of this round complete (first round: cursor as well)
      // 2c. ranks from the bit masks
      if ((int)threadIdx.x < nx) {                      // per tile column: running count over the mask words
        unsigned int run = cursor[threadIdx.x];
#pragma unroll 8
        for (int k = 0; k < RS_WORDS; ++k) { pref[k][threadIdx.x] = run; run += __popc(mask[k][threadIdx.x]); }
        cursor[threadIdx.x] = run;
      }
      __syncthreads();
      // 2d. ids to their final positions
      for (unsigned int hl = threadIdx.x; hl < m; hl += RS_THREADS) {
        const unsigned int id = ids[list_j[hl]], xw = list_x[hl], k = hl >> 5, below = (1u << (hl & 31)) - 1u;
        for (unsigned int x = xw & 0xffffu; x < (xw >> 16); ++x) pair_ids[pref[k][x] + __popc(mask[k][x] & below)] = id;
      }
    }
  }
}

__global__ void l1_loss_kernel(const float* __restrict__ image, const float* __restrict__ target, const long long count,
                               float* __restrict__ dL, float* loss, const unsigned int* __restrict__ overflow_flag) {
  const float inv = 1.0f / (float)count;
  float acc = 0.f;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
    const float d = image[i] - target[i];
    acc += fabsf(d);
    dL[i] = d > 0.f ? inv : (d < 0.f ? -inv : 0.f);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (overflow_flag && *overflow_flag) acc = __int_as_float(0x7fc00000);   // pair capacity exceeded: nothing was drawn
  if ((threadIdx.x & 31) == 0) atomicAdd(loss, acc * inv);
}

void launch_compact_and_tile_grid(const Workspace& ws, int N, int K, const ViewParams& vp, const CfgParams& cp, long long cap, cudaStream_t st) {
  const int blocks = N > 0 ? (N + SCAN_TILE - 1) / SCAN_TILE : 0;
  const size_t smem = 4 * (size_t)(vp.tiles_x + 1) * (vp.tiles_y + 1);
  cudaFuncSetAttribute(compact_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * MAX_GRID_CELLS);   // per device, cheap: every call
  WsHeader mirror{};
  mirror.N = N; mirror.K = K; mirror.W = vp.width; mirror.H = vp.height; mirror.pair_capacity = cap; mirror.tiles = (long long)vp.tiles_x * vp.tiles_y;
  compact_kernel<<<blocks + 1, SCAN_THREADS, smem, st>>>(ws.tiles_touched, ws.rec, N, ws.hdr, ws.scan_state[0], ws.l1_keys[0], ws.l1_vals[0], ws.vis_ids,
                                                        ws.sort_hist, ws.tile_diff, vp.tiles_x, vp.tiles_y, (unsigned int)cap, mirror, ws.ranges,
                                                        depth_key_base(cp));
  count_launch();
}

void launch_row_ballots(const Workspace& ws, int N, const ViewParams& vp, int num_sms, cudaStream_t st) {
  if (N <= 0) return;
  const long long warps = ((long long)N + 31) / 32, ctas = (warps + 7) / 8;       // the survivor count lives on the device: grid-stride over its iterations
  const int blocks = (int)(ctas < 8LL * num_sms ? ctas : 8LL * num_sms);
  row_ballot_kernel<<<blocks, 256, 0, st>>>(ws.hdr, ws.sorted_ys, vp.tiles_y, ws.rb_stride, ws.row_ballots);
  count_launch();
}

void launch_row_scatter(const Workspace& ws, int N, const ViewParams& vp, int num_sms, cudaStream_t st) {
  if (N <= 0) return;
  const int xblocks = (vp.tiles_x + RS_XB - 1) / RS_XB;
  // the survivor count lives on the device: persistent CTAs take (chunk, row, column block) items from a ticket
  const unsigned long long items = (unsigned long long)ws.rs_chunks * (unsigned int)vp.tiles_y * xblocks;
  const unsigned int blocks = (unsigned int)(items < 8ull * num_sms ? items : 8ull * num_sms);
  row_scatter_kernel<<<blocks, RS_THREADS, 0, st>>>(ws.hdr, ws.row_ballots, ws.rb_stride, ws.sorted_xs, ws.sorted_ids, ws.ranges, ws.rs_state, vp.tiles_x, vp.tiles_y,
                                                    xblocks, ws.rs_chunk, ws.pair_ids);
  count_launch();
}

void launch_l1_loss(const float* image, const float* target, long long count, float* dL, float* loss, const unsigned int* overflow_flag,
                    cudaStream_t st) {
  l1_loss_kernel<<<592, 256, 0, st>>>(image, target, count, dL, loss, overflow_flag);
  count_launch();
}

}  // namespace fdgs
