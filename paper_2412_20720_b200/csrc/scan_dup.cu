// scan_dup.cu — A5/A6/A7b/A8 for sm_100a: compaction scan (+ depth digit counts) with the tile-grid prefix (ranges, D) as a
// role of its first CTA, offsets scan, and the rectangle-aware ordered scatter that writes the per-tile lists.
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
  for (int i = threadIdx.x; i < cells; i += blockDim.x) grid[i] = tile_diff[i];
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
  for (int x = threadIdx.x; x < sx; x += blockDim.x) { int run = 0; for (int y = 0; y < rows; ++y) { run += grid[y * sx + x]; grid[y * sx + x] = run; } }
  __syncthreads();
  // exclusive scan over tiles in row-major order; each thread owns a contiguous chunk
  const int per = (tiles + blockDim.x - 1) / blockDim.x, t0 = threadIdx.x * per, t1 = min(t0 + per, tiles);
  unsigned int sum = 0;
  for (int t = t0; t < t1; ++t) sum += (unsigned int)grid[(t / tiles_x) * sx + (t % tiles_x)];
  unsigned int total;
  unsigned int run = block_exclusive_scan(sum, total, warp_sums);
  const bool overflow = total > cap;
  for (int t = t0; t < t1; ++t) {
    const unsigned int c = (unsigned int)grid[(t / tiles_x) * sx + (t % tiles_x)];
    ranges[t] = overflow ? make_uint2(0, 0) : make_uint2(run, run + c);
    run += c;
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
                                                               const WsHeader mirror, uint2* __restrict__ ranges) {
  extern __shared__ int grid[];                 // (tiles_y+1) x (tiles_x+1), used by CTA 0 only
  __shared__ unsigned int warp_sums[33], s_tile, s_prefix, hist[4][RADIX];
  if (blockIdx.x == 0) { tile_grid_role(tile_diff, tiles_x, tiles_y, cap, hdr, mirror, ranges, grid, warp_sums); return; }
  if (threadIdx.x == 0) s_tile = atomicAdd(&hdr->scan_ticket[0], 1u);
#pragma unroll
  for (int p = 0; p < 4; ++p) hist[p][threadIdx.x] = 0;     // SCAN_THREADS == RADIX
  __syncthreads();
  const unsigned int tile = s_tile;
  const long long base = (long long)tile * SCAN_TILE + (long long)threadIdx.x * SCAN_ITEMS;
  unsigned int flags = 0, cnt = 0;
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
      const unsigned int key = __float_as_uint(rec[base + k].depth);
      keys[pos] = key; vals[pos] = (unsigned int)(base + k); vis_ids[pos] = (unsigned int)(base + k); ++pos;
#pragma unroll
      for (int p = 0; p < 4; ++p) atomicAdd(&hist[p][(key >> (RADIX_BITS * p)) & (RADIX - 1)], 1u);
    }
  if (tile == gridDim.x - 2 && threadIdx.x == 0) hdr->num_visible = prefix + total;    // gridDim.x - 1 compaction tiles
  __syncthreads();
#pragma unroll
  for (int p = 0; p < 4; ++p) { const unsigned int v = hist[p][threadIdx.x]; if (v) atomicAdd(sort_hist + p * RADIX + threadIdx.x, v); }
}

// offsets[j] = exclusive prefix of tiles_touched[sorted_ids[j]], j < num_visible (depth order).  Also cuts the emission
// order into chunks of ~chunk_pairs pairs made of WHOLE survivors: survivor j belongs to chunk offsets[j] / chunk_pairs, and
// chunk_first[q] = the first survivor of chunk q or later (= num_visible past the last one), q <= num_chunks.
__global__ void __launch_bounds__(SCAN_THREADS) offsets_kernel(const unsigned int* __restrict__ tiles_touched,
                                                               const unsigned int* __restrict__ sorted_ids, WsHeader* hdr,
                                                               unsigned long long* state, unsigned int* __restrict__ offsets,
                                                               unsigned int* __restrict__ chunk_first, const unsigned int chunk_pairs,
                                                               const unsigned int num_chunks) {
  __shared__ unsigned int warp_sums[33], s_tile, s_prefix;
  const unsigned int n = hdr->num_visible;
  if (threadIdx.x == 0) s_tile = atomicAdd(&hdr->scan_ticket[1], 1u);
  __syncthreads();
  const unsigned int tile = s_tile;
  if (n == 0) {                                             // nothing visible: every chunk is empty
    if (tile == 0) for (unsigned int q = threadIdx.x; q <= num_chunks; q += blockDim.x) chunk_first[q] = 0;
    return;
  }
  if ((unsigned long long)tile * SCAN_TILE >= n) return;   // tickets are dense: every tile below this one exists
  const unsigned int base = tile * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  unsigned int c[SCAN_ITEMS], sum = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { c[k] = base + k < n ? tiles_touched[sorted_ids[base + k]] : 0; sum += c[k]; }
  unsigned int total;
  const unsigned int excl = block_exclusive_scan(sum, total, warp_sums);
  const unsigned int prefix = lookback_prefix(state, tile, total, &s_prefix);
  if (hdr->overflow) return;                               // D exceeds the capacity: nothing is emitted
  unsigned int run = prefix + excl;
  // chunk of the previous survivor (-1 before the first one): every chunk id in (previous, mine] starts at me
  long long prev_chunk = -1;
  if (base > 0 && base < n) prev_chunk = (long long)((run - tiles_touched[sorted_ids[base - 1]]) / chunk_pairs);
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    if (base + k < n) {
      offsets[base + k] = run;
      const long long mine = run / chunk_pairs;
      for (long long q = prev_chunk + 1; q <= mine; ++q) chunk_first[q] = base + k;
      prev_chunk = mine;
      if (base + k == n - 1) for (unsigned int q = (unsigned int)mine + 1; q <= num_chunks; ++q) chunk_first[q] = n;
    }
    run += c[k];
  }
}

// ---------------------------------------------------------------------------------------------
// A6/A7, level 2: the per-tile lists in depth order, written straight to their final place.
//
// Survivors arrive sorted by depth (level 1); survivor j covers the tile rectangle rect[j].  The list of tile T is
// {j : T in rect[j]} in ascending j, stored at [ranges[T].x, ranges[T].y) — a stable partition of the emission order
// (j, tiles of rect[j]) by tile, i.e. what a stable sort of the (tile, id) pairs by tile id produces.  Because the ranges
// are already known from the coverage grid and the covered sets are RECTANGLES, no sort is needed:
//   1. chunk_cover_kernel: the emission order is cut into chunks of whole survivors (chunk_first); a CTA builds the
//      coverage count of its chunk for every tile with a 2D difference array in shared memory (4 atomics per survivor +
//      one 2D prefix, whatever the footprints);
//   2. chunk_base_kernel: exclusive prefix over the chunks, per tile, started at ranges[T].x = the output position at
//      which chunk q starts writing in tile T;
//   3. pair_scatter_kernel: a CTA per chunk walks its survivors in order, 32 at a time.  Within such a group the
//      rank of survivor s in tile T is the number of lower-numbered members that also cover T: every (member, tile)
//      pair ORs its member bit into a per-tile mask in shared memory, the rank is a popcount of the lower bits, and the
//      highest member advances the tile's cursor by the group's count.  O(1) work per pair, 4 bytes written per pair,
//      no key array, no look-back, no histogram.
// Replaces offsets + pair emission + a 2-pass radix sort of the D pairs (round 1: 146 us per view at cfg3).
__global__ void __launch_bounds__(256) chunk_cover_kernel(const unsigned int* __restrict__ sorted_ids, const ushort4* __restrict__ rect,
                                                          const WsHeader* __restrict__ hdr, const unsigned int* __restrict__ chunk_first,
                                                          const unsigned int chunk_pairs, const int tiles_x, const int tiles_y,
                                                          unsigned int* __restrict__ chunk_base) {
  extern __shared__ int grid[];                 // (tiles_y+1) x (tiles_x+1)
  const unsigned int D = hdr->num_pairs;
  const unsigned int q = blockIdx.x;
  if ((unsigned long long)q * chunk_pairs >= D) return;    // also covers overflow (num_pairs == 0)
  const int sx = tiles_x + 1, rows = tiles_y + 1, cells = sx * rows;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  for (int i = threadIdx.x; i < cells; i += blockDim.x) grid[i] = 0;
  __syncthreads();
  const unsigned int j0 = chunk_first[q], j1 = chunk_first[q + 1];
  for (unsigned int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
    const ushort4 rc = rect[sorted_ids[j]];
    atomicAdd(&grid[rc.y * sx + rc.x], 1); atomicAdd(&grid[rc.y * sx + rc.z], -1);
    atomicAdd(&grid[rc.w * sx + rc.x], -1); atomicAdd(&grid[rc.w * sx + rc.z], 1);
  }
  __syncthreads();
  for (int y = warp; y < rows; y += nwarps) {
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
  // column pass fused with the write-out: thread x walks down its column
  unsigned int* out = chunk_base + (size_t)q * tiles_x * tiles_y;
  for (int x = threadIdx.x; x < tiles_x; x += blockDim.x) {
    int run = 0;
    for (int y = 0; y < tiles_y; ++y) { run += grid[y * sx + x]; out[y * tiles_x + x] = (unsigned int)run; }
  }
}

// exclusive prefix over the active chunks, per tile, in place; thread (g, t): chunk group g of CB_GROUPS, tile t of 32
constexpr int CB_GROUPS = 8, CB_TILES = 32;
__global__ void __launch_bounds__(CB_GROUPS * CB_TILES) chunk_base_kernel(const WsHeader* __restrict__ hdr, const uint2* __restrict__ ranges,
                                                                            const unsigned int chunk_pairs, const int tiles,
                                                                            unsigned int* __restrict__ chunk_base) {
  __shared__ unsigned int part[CB_GROUPS][CB_TILES];
  const unsigned int D = hdr->num_pairs;
  if (D == 0) return;
  const unsigned int nq = (D + chunk_pairs - 1) / chunk_pairs;         // active chunks
  const int t = blockIdx.x * CB_TILES + (threadIdx.x & (CB_TILES - 1)), g = threadIdx.x / CB_TILES;
  const unsigned int per = (nq + CB_GROUPS - 1) / CB_GROUPS, q0 = min(nq, g * per), q1 = min(nq, q0 + per);
  unsigned int sum = 0;
  if (t < tiles) for (unsigned int q = q0; q < q1; ++q) sum += chunk_base[(size_t)q * tiles + t];
  part[g][threadIdx.x & (CB_TILES - 1)] = sum;
  __syncthreads();
  if (t >= tiles) return;
  unsigned int run = ranges[t].x;
  for (int gg = 0; gg < g; ++gg) run += part[gg][threadIdx.x & (CB_TILES - 1)];
  for (unsigned int q = q0; q < q1; ++q) { const size_t i = (size_t)q * tiles + t; const unsigned int c = chunk_base[i]; chunk_base[i] = run; run += c; }
}

constexpr int SC_GROUP = 32;        // survivors ranked together (one bit each in the per-tile mask)
constexpr int SC_STAGE = 1024;      // survivors staged in shared memory at a time
template <bool CURSOR_SMEM>
__global__ void __launch_bounds__(256) pair_scatter_kernel(const unsigned int* __restrict__ sorted_ids, const unsigned int* __restrict__ offsets,
                                                           const ushort4* __restrict__ rect, const WsHeader* __restrict__ hdr,
                                                           const unsigned int* __restrict__ chunk_first, const unsigned int chunk_pairs,
                                                           const int tiles_x, const int tiles, unsigned int* __restrict__ chunk_base,
                                                           unsigned int* __restrict__ pair_ids) {
  extern __shared__ unsigned int sc_smem[];     // mask[tiles] (+ cursor[tiles] if CURSOR_SMEM)
  __shared__ unsigned int s_off[SC_STAGE + 1], s_id[SC_STAGE];
  __shared__ ushort4 s_rc[SC_STAGE];
  const unsigned int D = hdr->num_pairs;
  const unsigned int q = blockIdx.x;
  if ((unsigned long long)q * chunk_pairs >= D) return;
  unsigned int* mask = sc_smem;
  unsigned int* cursor = CURSOR_SMEM ? sc_smem + tiles : chunk_base + (size_t)q * tiles;
  for (int i = threadIdx.x; i < tiles; i += blockDim.x) { mask[i] = 0; if (CURSOR_SMEM) cursor[i] = chunk_base[(size_t)q * tiles + i]; }
  const unsigned int j0 = chunk_first[q], j1 = chunk_first[q + 1];
  for (unsigned int jb = j0; jb < j1; jb += SC_STAGE) {
    const unsigned int m = min((unsigned int)SC_STAGE, j1 - jb);
    __syncthreads();                                      // previous stage consumed; (first trip) mask / cursor initialised
    for (unsigned int s = threadIdx.x; s < m; s += blockDim.x) {
      const unsigned int id = sorted_ids[jb + s];
      s_off[s] = offsets[jb + s]; s_id[s] = id; s_rc[s] = rect[id];
    }
    __syncthreads();
    if (threadIdx.x == 0) { const ushort4 rc = s_rc[m - 1]; s_off[m] = s_off[m - 1] + (unsigned int)(rc.z - rc.x) * (unsigned int)(rc.w - rc.y); }
    __syncthreads();
    for (unsigned int g0 = 0; g0 < m; g0 += SC_GROUP) {   // groups of 32 survivors, in order
      const unsigned int gm = min((unsigned int)SC_GROUP, m - g0);
      const unsigned int e0 = s_off[g0], e1 = s_off[g0 + gm];
      // a thread owns the pairs e0 + tid + 256 i; the first PC of them keep (tile, member) in registers across the phases
      constexpr int PC = 4;
      unsigned int ctile[PC], cbit[PC];
      auto locate = [&](const unsigned int e, unsigned int& tile, unsigned int& bit) {
        unsigned int lo = g0, hi = g0 + gm;                // largest s with s_off[s] <= e
        while (hi - lo > 1) { const unsigned int mid = (lo + hi) >> 1; if (s_off[mid] <= e) lo = mid; else hi = mid; }
        const ushort4 rc = s_rc[lo];
        const unsigned int local = e - s_off[lo], w = rc.z - rc.x;
        tile = (rc.y + local / w) * tiles_x + rc.x + local % w;
        bit = lo - g0;
      };
      // phase 1: every pair of the group finds its member and tile, and sets its bit in the tile's mask
#pragma unroll
      for (int i = 0; i < PC; ++i) {
        const unsigned int e = e0 + threadIdx.x + i * 256;
        if (e < e1) { locate(e, ctile[i], cbit[i]); atomicOr(&mask[ctile[i]], 1u << cbit[i]); }
      }
      for (unsigned int e = e0 + threadIdx.x + PC * 256; e < e1; e += 256) { unsigned int t, b; locate(e, t, b); atomicOr(&mask[t], 1u << b); }
      __syncthreads();
      // phase 2: rank inside the group = members below me that cover the tile; the cursor is not touched yet
#pragma unroll
      for (int i = 0; i < PC; ++i) {
        const unsigned int e = e0 + threadIdx.x + i * 256;
        if (e < e1) pair_ids[cursor[ctile[i]] + __popc(mask[ctile[i]] & ((1u << cbit[i]) - 1u))] = s_id[g0 + cbit[i]];
      }
      for (unsigned int e = e0 + threadIdx.x + PC * 256; e < e1; e += 256) {
        unsigned int t, b; locate(e, t, b);
        pair_ids[cursor[t] + __popc(mask[t] & ((1u << b) - 1u))] = s_id[g0 + b];
      }
      __syncthreads();
      // phase 3: the highest member of a tile advances its cursor by the group's count and clears the mask
#pragma unroll
      for (int i = 0; i < PC; ++i) {
        const unsigned int e = e0 + threadIdx.x + i * 256;
        if (e < e1) { const unsigned int mk = mask[ctile[i]]; if ((mk >> cbit[i]) == 1u) { cursor[ctile[i]] += __popc(mk); mask[ctile[i]] = 0; } }
      }
      for (unsigned int e = e0 + threadIdx.x + PC * 256; e < e1; e += 256) {
        unsigned int t, b; locate(e, t, b);
        const unsigned int mk = mask[t];
        if ((mk >> b) == 1u) { cursor[t] += __popc(mk); mask[t] = 0; }
      }
      __syncthreads();
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

void launch_compact_and_tile_grid(const Workspace& ws, int N, int K, const ViewParams& vp, long long cap, cudaStream_t st) {
  const int blocks = N > 0 ? (N + SCAN_TILE - 1) / SCAN_TILE : 0;
  const size_t smem = 4 * (size_t)(vp.tiles_x + 1) * (vp.tiles_y + 1);
  static bool attr_set = false;
  if (!attr_set) { cudaFuncSetAttribute(compact_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * MAX_GRID_CELLS); attr_set = true; }
  WsHeader mirror{};
  mirror.N = N; mirror.K = K; mirror.W = vp.width; mirror.H = vp.height; mirror.pair_capacity = cap; mirror.tiles = (long long)vp.tiles_x * vp.tiles_y;
  compact_kernel<<<blocks + 1, SCAN_THREADS, smem, st>>>(ws.tiles_touched, ws.rec, N, ws.hdr, ws.scan_state[0], ws.l1_keys[0], ws.l1_vals[0], ws.vis_ids,
                                                        ws.sort_hist, ws.tile_diff, vp.tiles_x, vp.tiles_y, (unsigned int)cap, mirror, ws.ranges);
  count_launch();
}

void launch_offsets(const Workspace& ws, int l1_buf, int N, cudaStream_t st) {
  if (N <= 0) return;
  const int blocks = (N + SCAN_TILE - 1) / SCAN_TILE;
  offsets_kernel<<<blocks, SCAN_THREADS, 0, st>>>(ws.tiles_touched, ws.l1_vals[l1_buf], ws.hdr, ws.scan_state[1], ws.offsets, ws.chunk_first,
                                                  ws.chunk_pairs, ws.num_chunks);
  count_launch();
}

void launch_pair_scatter(const Workspace& ws, int l1_buf, int N, const ViewParams& vp, int num_sms, cudaStream_t st) {
  if (N <= 0) return;
  (void)num_sms;
  const int tiles = vp.tiles_x * vp.tiles_y;
  const size_t grid_smem = 4 * (size_t)(vp.tiles_x + 1) * (vp.tiles_y + 1);
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(chunk_cover_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * MAX_GRID_CELLS);
    cudaFuncSetAttribute(pair_scatter_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 8 * (MAX_GRID_CELLS / 2));
    cudaFuncSetAttribute(pair_scatter_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * MAX_GRID_CELLS);
    attr_set = true;
  }
  // D lives on the device: one CTA per possible chunk of the capacity, surplus CTAs exit at once
  chunk_cover_kernel<<<ws.num_chunks, 256, grid_smem, st>>>(ws.l1_vals[l1_buf], ws.rect, ws.hdr, ws.chunk_first, ws.chunk_pairs, vp.tiles_x, vp.tiles_y, ws.chunk_base);
  chunk_base_kernel<<<(tiles + CB_TILES - 1) / CB_TILES, CB_GROUPS * CB_TILES, 0, st>>>(ws.hdr, ws.ranges, ws.chunk_pairs, tiles, ws.chunk_base);
  if (tiles <= MAX_GRID_CELLS / 2)
    pair_scatter_kernel<true><<<ws.num_chunks, 256, 8 * (size_t)tiles, st>>>(ws.l1_vals[l1_buf], ws.offsets, ws.rect, ws.hdr, ws.chunk_first, ws.chunk_pairs,
                                                                           vp.tiles_x, tiles, ws.chunk_base, ws.pair_ids);
  else
    pair_scatter_kernel<false><<<ws.num_chunks, 256, 4 * (size_t)tiles, st>>>(ws.l1_vals[l1_buf], ws.offsets, ws.rect, ws.hdr, ws.chunk_first, ws.chunk_pairs,
                                                                            vp.tiles_x, tiles, ws.chunk_base, ws.pair_ids);
  count_launch(3);
}

void launch_l1_loss(const float* image, const float* target, long long count, float* dL, float* loss, const unsigned int* overflow_flag,
                    cudaStream_t st) {
  l1_loss_kernel<<<592, 256, 0, st>>>(image, target, count, dL, loss, overflow_flag);
  count_launch();
}

}  // namespace fdgs
