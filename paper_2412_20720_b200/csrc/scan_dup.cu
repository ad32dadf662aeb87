// scan_dup.cu — A5/A6/A8 for sm_100a: compaction scan (+ depth digit counts), tile-grid prefix (ranges, D), offsets scan, pair emission.
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

// Compaction: survivors (tiles_touched > 0) in primitive-id order -> (depth bits, id) pairs, plus the digit counts of
// the four 8-bit passes of the depth sort (the keys are in registers here: the sort never reads them just to count).
__global__ void __launch_bounds__(SCAN_THREADS) compact_kernel(const unsigned int* __restrict__ tiles_touched,
                                                               const SplatRec* __restrict__ rec, const int N, WsHeader* hdr,
                                                               unsigned long long* state, unsigned int* __restrict__ keys,
                                                               unsigned int* __restrict__ vals, unsigned int* __restrict__ vis_ids,
                                                               unsigned int* __restrict__ sort_hist) {
  __shared__ unsigned int warp_sums[33], s_tile, s_prefix, hist[4][RADIX];
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
  if (tile == gridDim.x - 1 && threadIdx.x == 0) hdr->num_visible = prefix + total;
  __syncthreads();
#pragma unroll
  for (int p = 0; p < 4; ++p) { const unsigned int v = hist[p][threadIdx.x]; if (v) atomicAdd(sort_hist + p * RADIX + threadIdx.x, v); }
}

// offsets[j] = exclusive prefix of tiles_touched[sorted_ids[j]], j < num_visible (depth order).  Also fills the table the pair
// emission starts from: chunk_first[k] = the survivor whose pairs contain output position k * DUP_CHUNK.
__global__ void __launch_bounds__(SCAN_THREADS) offsets_kernel(const unsigned int* __restrict__ tiles_touched,
                                                               const unsigned int* __restrict__ sorted_ids, WsHeader* hdr,
                                                               unsigned long long* state, unsigned int* __restrict__ offsets,
                                                               unsigned int* __restrict__ chunk_first) {
  __shared__ unsigned int warp_sums[33], s_tile, s_prefix;
  const unsigned int n = hdr->num_visible;
  if (threadIdx.x == 0) s_tile = atomicAdd(&hdr->scan_ticket[1], 1u);
  __syncthreads();
  const unsigned int tile = s_tile;
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
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    if (base + k < n) {
      offsets[base + k] = run;
      for (unsigned int q = (run + DUP_CHUNK - 1) / DUP_CHUNK; q * DUP_CHUNK < run + c[k]; ++q) chunk_first[q] = base + k;
    }
    run += c[k];
  }
}

// ---------------------------------------------------------------------------------------------
// Tile grid: 2D inclusive prefix of the coverage difference array = list length of every tile; its
// exclusive scan in tile order = the tile ranges (A8) and D; digit histograms of the tile ids weighted
// by list length = the global digit bases of the level-2 radix passes.  One CTA, all in shared memory.
__global__ void __launch_bounds__(1024) tile_grid_kernel(const int* __restrict__ tile_diff, const int tiles_x, const int tiles_y,
                                                         const unsigned int cap, const int l2_passes, WsHeader* hdr,
                                                         uint2* __restrict__ ranges, unsigned int* __restrict__ sort_hist) {
  extern __shared__ int grid[];                 // (tiles_y+1) x (tiles_x+1)
  __shared__ unsigned int warp_sums[33], hist[4][RADIX];
  const int sx = tiles_x + 1, cells = sx * (tiles_y + 1), tiles = tiles_x * tiles_y;
  for (int i = threadIdx.x; i < cells; i += blockDim.x) grid[i] = tile_diff[i];
  for (int i = threadIdx.x; i < 4 * RADIX; i += blockDim.x) (&hist[0][0])[i] = 0;
  __syncthreads();
  for (int y = threadIdx.x; y <= tiles_y; y += blockDim.x) { int run = 0; for (int x = 0; x < sx; ++x) { run += grid[y * sx + x]; grid[y * sx + x] = run; } }
  __syncthreads();
  for (int x = threadIdx.x; x < sx; x += blockDim.x) { int run = 0; for (int y = 0; y <= tiles_y; ++y) { run += grid[y * sx + x]; grid[y * sx + x] = run; } }
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
    if (c)
      for (int p = 0; p < l2_passes; ++p) atomicAdd(&hist[p][(t >> (RADIX_BITS * p)) & (RADIX - 1)], c);
  }
  __syncthreads();
  // exclusive digit bases per pass (RADIX == 256 <= blockDim): warps 0..7 scan one pass's 256 bins, 8 per lane
  if (threadIdx.x < 32 * l2_passes) {
    const int p = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned int v[8], s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) { v[k] = hist[p][lane * 8 + k]; s += v[k]; }
    unsigned int incl = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned int n = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += n; }
    unsigned int r = incl - s;
#pragma unroll
    for (int k = 0; k < 8; ++k) { sort_hist[(4 + p) * RADIX + lane * 8 + k] = r; r += v[k]; }
  }
  if (threadIdx.x == 0) { hdr->num_pairs = overflow ? 0u : total; hdr->overflow = overflow ? 1u : 0u; hdr->pad[0] = total; }
}

// ---------------------------------------------------------------------------------------------
// A6: pair emission in depth order, balanced by OUTPUT: a CTA owns DUP_CHUNK consecutive pairs whatever the footprints of
// the survivors that produce them (a splat covering the whole screen is spread over many CTAs, thousands of one-tile
// splats share one).  The survivors of the chunk [chunk_first[k], chunk_first[k+1]] are staged in shared memory (offset,
// id, rectangle), every thread finds the owner of its pairs by binary search there, and all stores are coalesced.
__global__ void __launch_bounds__(256) duplicate_kernel(const unsigned int* __restrict__ sorted_ids, const unsigned int* __restrict__ offsets,
                                                        const ushort4* __restrict__ rect, const WsHeader* __restrict__ hdr,
                                                        const unsigned int* __restrict__ chunk_first, const int tiles_x,
                                                        unsigned int* __restrict__ keys, unsigned int* __restrict__ vals) {
  __shared__ unsigned int s_off[DUP_CHUNK + 1], s_id[DUP_CHUNK + 1];
  __shared__ ushort4 s_rc[DUP_CHUNK + 1];
  const unsigned int D = hdr->num_pairs, n = hdr->num_visible;
  const unsigned int start = blockIdx.x * DUP_CHUNK;
  if (start >= D) return;                                  // also covers overflow (num_pairs == 0)
  const unsigned int end = min(start + DUP_CHUNK, D);
  const unsigned int j0 = chunk_first[blockIdx.x];
  const unsigned int j1 = end < D ? chunk_first[blockIdx.x + 1] : n - 1;     // last survivor with pairs in this chunk
  const unsigned int m = j1 - j0 + 1;                      // <= DUP_CHUNK + 1: every survivor emits at least one pair
  for (unsigned int s = threadIdx.x; s < m; s += blockDim.x) {
    const unsigned int id = sorted_ids[j0 + s];
    s_off[s] = offsets[j0 + s]; s_id[s] = id; s_rc[s] = rect[id];
  }
  __syncthreads();
  for (unsigned int e = start + threadIdx.x; e < end; e += blockDim.x) {
    unsigned int lo = 0, hi = m;                           // largest s with s_off[s] <= e
    while (hi - lo > 1) { const unsigned int mid = (lo + hi) >> 1; if (s_off[mid] <= e) lo = mid; else hi = mid; }
    const ushort4 rc = s_rc[lo];
    const unsigned int local = e - s_off[lo], w = rc.z - rc.x;
    keys[e] = (rc.y + local / w) * tiles_x + rc.x + local % w;
    vals[e] = s_id[lo];
  }
}

__global__ void l1_loss_kernel(const float* __restrict__ image, const float* __restrict__ target, const long long count,
                               float* __restrict__ dL, float* loss) {
  const float inv = 1.0f / (float)count;
  float acc = 0.f;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
    const float d = image[i] - target[i];
    acc += fabsf(d);
    dL[i] = d > 0.f ? inv : (d < 0.f ? -inv : 0.f);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) atomicAdd(loss, acc * inv);
}

void launch_compact(const Workspace& ws, int N, cudaStream_t st) {
  if (N <= 0) return;
  const int blocks = (N + SCAN_TILE - 1) / SCAN_TILE;
  compact_kernel<<<blocks, SCAN_THREADS, 0, st>>>(ws.tiles_touched, ws.rec, N, ws.hdr, ws.scan_state[0], ws.l1_keys[0], ws.l1_vals[0], ws.vis_ids, ws.sort_hist);
  ++g_launches;
}

void launch_offsets(const Workspace& ws, int l1_buf, int N, cudaStream_t st) {
  if (N <= 0) return;
  const int blocks = (N + SCAN_TILE - 1) / SCAN_TILE;
  offsets_kernel<<<blocks, SCAN_THREADS, 0, st>>>(ws.tiles_touched, ws.l1_vals[l1_buf], ws.hdr, ws.scan_state[1], ws.offsets, ws.chunk_first);
  ++g_launches;
}

void launch_tile_grid(const Workspace& ws, const ViewParams& vp, long long cap, int l2_passes, cudaStream_t st) {
  const size_t smem = 4 * (size_t)(vp.tiles_x + 1) * (vp.tiles_y + 1);
  static bool attr_set = false;
  if (!attr_set) { cudaFuncSetAttribute(tile_grid_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * MAX_GRID_CELLS); attr_set = true; }
  tile_grid_kernel<<<1, 1024, smem, st>>>(ws.tile_diff, vp.tiles_x, vp.tiles_y, (unsigned int)cap, l2_passes, ws.hdr, ws.ranges, ws.sort_hist);
  ++g_launches;
}

void launch_duplicate(const Workspace& ws, int l1_buf, int N, long long cap, const ViewParams& vp, cudaStream_t st) {
  if (N <= 0) return;
  // D lives on the device: one CTA per possible chunk of the capacity, surplus CTAs exit at once
  const unsigned int blocks = (unsigned int)((cap + DUP_CHUNK - 1) / DUP_CHUNK);
  duplicate_kernel<<<blocks, 256, 0, st>>>(ws.l1_vals[l1_buf], ws.offsets, ws.rect, ws.hdr, ws.chunk_first, vp.tiles_x, ws.l2_keys[0], ws.l2_vals[0]);
  ++g_launches;
}

void launch_l1_loss(const float* image, const float* target, long long count, float* dL, float* loss, cudaStream_t st) {
  l1_loss_kernel<<<592, 256, 0, st>>>(image, target, count, dL, loss);
  ++g_launches;
}

}  // namespace fdgs
