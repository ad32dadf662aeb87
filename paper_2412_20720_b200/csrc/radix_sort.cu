// radix_sort.cu — A7: hand-written stable LSD radix sort of (u32 key, u32 value) pairs for sm_100a.
// One kernel per 9-bit digit ("onesweep"): each CTA ranks a tile of pairs in shared memory with warp-level
// ballot-per-bit multisplit (stable; MATCH.ANY measured 14 % slower: it loops once per distinct digit), publishes its digit counts, obtains the counts of all earlier tiles by
// decoupled look-back, and scatters straight to the final position of the pass — keys and values are read
// once and written once per pass.  Tiles take dynamic ids from a ticket, CTAs are persistent, and the number
// of pairs is read from device memory, so the host never synchronises.  The global digit counts come from the producer
// of the keys (the compaction kernel): the keys are never read just to be counted.  Since round 2 only the depth sort of
// the survivors (level 1) is a radix sort; the (tile, id) pairs are placed by the ordered scatter of scan_dup.cu.
#include "common.cuh"

namespace fdgs {

constexpr int LB_WIN = 8;
constexpr unsigned int LB_AGG = 1u << 30, LB_PRE = 2u << 30, LB_MASK = (1u << 30) - 1;

// MODE 0: a pass that always runs.  MODE 1: the third pass — the last one unless a key has bits above 3 RADIX_BITS, in which
// case the fourth (MODE 2) is; whichever is last also writes the ids and the tile rectangles of the survivors in the
// final order (ys = y0 | y1 << 16, xs = x0 | x1 << 16: the row scatter reads them coalesced).  The decision is the digit
// count top_zero = sort_hist[3][0] (keys whose fourth digit is zero) against the number of survivors: no host round trip.
// A thread owns the digits 2t and 2t + 1: their counts, look-back words (one 64-bit word per pair, published and read
// whole) and bases.
// 3 CTAs per SM (<= 85 registers): measured best at 50 M pairs (812 us for two passes vs 916 us at 2 CTAs / 128 registers);
// 4 or 5 CTAs spill.
template <int ITEMS, int MODE>
__global__ void __launch_bounds__(SORT_THREADS, 3) onesweep_kernel(const unsigned int* __restrict__ keys_in, const unsigned int* __restrict__ vals_in,
                                                                unsigned int* __restrict__ keys_out, unsigned int* __restrict__ vals_out,
                                                                const unsigned int* __restrict__ count_dev, unsigned int* ticket,
                                                                const unsigned int* __restrict__ digit_count /*[RADIX] raw counts of this pass*/,
                                                                const unsigned int* __restrict__ top_zero, volatile unsigned long long* lookback,
                                                                const int shift, const ushort4* __restrict__ rect, unsigned int* __restrict__ ys_out,
                                                                unsigned int* __restrict__ xs_out, unsigned int* __restrict__ ids_out) {
  constexpr int TILE_N = SORT_THREADS * ITEMS, WARPS = SORT_THREADS / 32;
  __shared__ __align__(16) unsigned int warp_hist[WARPS][RADIX];   // per-warp digit counts -> exclusive offsets over warps
  __shared__ __align__(16) unsigned int s_local[RADIX];            // first slot of each digit inside the sorted tile
  __shared__ __align__(16) unsigned int s_global[RADIX];           // global position of that slot (minus the slot index)
  __shared__ unsigned int s_keys[TILE_N], s_vals[TILE_N];
  __shared__ unsigned int warp_sums[33], s_tile;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned int lt_mask = (1u << lane) - 1;
  const unsigned int n = *count_dev;
  const bool fourth_needed = MODE != 0 && *top_zero != n;
  if (MODE == 2 && !fourth_needed) return;            // every key fits the first three digits: the third pass was the last
  const bool gather = MODE == 2 || (MODE == 1 && !fourth_needed);
  const unsigned int num_tiles = (n + TILE_N - 1) / TILE_N;
  // global position of the first key of the digits 2t, 2t + 1: exclusive scan of the raw digit counts
  unsigned int my_base[2];
  {
    const uint2 c = reinterpret_cast<const uint2*>(digit_count)[threadIdx.x];
    unsigned int incl = c.x + c.y;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
    if (lane == 31) warp_sums[warp] = incl;
    __syncthreads();
    unsigned int wprefix = 0;
#pragma unroll
    for (int w = 0; w < WARPS; ++w) if (w < warp) wprefix += warp_sums[w];
    my_base[0] = wprefix + incl - (c.x + c.y);
    my_base[1] = my_base[0] + c.x;
    __syncthreads();
  }
  while (true) {
    if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
#pragma unroll
    for (int w = 0; w < WARPS; ++w) { warp_hist[w][threadIdx.x] = 0; warp_hist[w][threadIdx.x + SORT_THREADS] = 0; }
    __syncthreads();
    const unsigned int tile = s_tile;
    if (tile >= num_tiles) break;
    // ---- load: warp w owns the contiguous chunk [w*32*ITEMS, (w+1)*32*ITEMS) of the tile, round r = 32 consecutive pairs
    const unsigned int tile_base = tile * TILE_N, warp_base = tile_base + warp * 32 * ITEMS;
    unsigned int key[ITEMS], val[ITEMS];
    unsigned short rank[ITEMS];
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
      const unsigned int idx = warp_base + r * 32 + lane;
      key[r] = idx < n ? keys_in[idx] : 0xffffffffu;
      val[r] = idx < n ? vals_in[idx] : 0u;
    }
    // ---- stable rank inside the warp's chunk: ballots over the digit bits group equal digits; the lowest lane of a group adds the group
    // size to the warp's digit counter with one shared atomic that returns the count of earlier rounds.  The ITEMS
    // peer masks are independent of each other and the atomics of one warp retire in program order, so nothing in this
    // loop waits on the previous round.
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
      const bool valid = warp_base + r * 32 + lane < n;
      const unsigned int digit = valid ? ((key[r] >> shift) & (RADIX - 1)) : 0xffffffffu;
      // peers with the same digit by one ballot per digit bit: MATCH.ANY loops in hardware once per DISTINCT value in the
      // warp, and the digits of 32 neighbouring pairs are almost always distinct here
      unsigned int peers = __ballot_sync(0xffffffffu, valid);
      if (!valid) peers = ~peers;
#pragma unroll
      for (int b = 0; b < RADIX_BITS; ++b) {
        const bool bit = (digit >> b) & 1u;
        const unsigned int bal = __ballot_sync(0xffffffffu, bit);
        peers &= bit ? bal : ~bal;
      }
      const int leader = __ffs(peers) - 1;
      unsigned int old = 0;
      if (valid && lane == leader) old = atomicAdd(&warp_hist[warp][digit], (unsigned int)__popc(peers));
      old = __shfl_sync(0xffffffffu, old, leader);
      rank[r] = (unsigned short)(old + __popc(peers & lt_mask));
    }
    __syncthreads();
    // ---- thread t owns the digits 2t, 2t + 1: exclusive offsets over warps, tile counts, look-back, local digit bases
    const int d0 = 2 * threadIdx.x;
    unsigned int cnt[2] = {0u, 0u};
#pragma unroll
    for (int w = 0; w < WARPS; ++w) {
      const uint2 c = *reinterpret_cast<uint2*>(&warp_hist[w][d0]);
      *reinterpret_cast<uint2*>(&warp_hist[w][d0]) = make_uint2(cnt[0], cnt[1]);
      cnt[0] += c.x; cnt[1] += c.y;
    }
    volatile unsigned long long* lb = lookback + (size_t)tile * (RADIX / 2) + threadIdx.x;
    const unsigned int flag0 = tile == 0 ? LB_PRE : LB_AGG;
    *lb = (unsigned long long)(flag0 | cnt[0]) | ((unsigned long long)(flag0 | cnt[1]) << 32);
    unsigned int excl_tiles[2] = {0u, 0u};
    if (tile > 0) {
      // windowed look-back: LB_WIN predecessors are read with independent loads, then consumed nearest first; the walk
      // stops at the first inclusive prefix and re-polls from the first entry that is not published yet
      long long j = (long long)tile - 1;
      bool found = false;
      while (!found) {
        unsigned long long sv[LB_WIN];
#pragma unroll
        for (int w = 0; w < LB_WIN; ++w) sv[w] = j - w >= 0 ? lookback[(size_t)(j - w) * (RADIX / 2) + threadIdx.x] : (((unsigned long long)LB_PRE << 32) | LB_PRE);
#pragma unroll
        for (int w = 0; w < LB_WIN; ++w) {
          const unsigned int lo = (unsigned int)sv[w], hi = (unsigned int)(sv[w] >> 32);
          if (found || (lo >> 30) == 0) break;
          excl_tiles[0] += lo & LB_MASK; excl_tiles[1] += hi & LB_MASK;
          --j;
          if ((lo >> 30) == 2) found = true;
        }
      }
      *lb = (unsigned long long)(LB_PRE | (excl_tiles[0] + cnt[0])) | ((unsigned long long)(LB_PRE | (excl_tiles[1] + cnt[1])) << 32);
    }
    // block exclusive scan of the counts over the 512 digits
    unsigned int incl = cnt[0] + cnt[1];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
    if (lane == 31) warp_sums[warp] = incl;
    __syncthreads();
    unsigned int wprefix = 0;
#pragma unroll
    for (int w = 0; w < WARPS; ++w) if (w < warp) wprefix += warp_sums[w];
    const unsigned int local0 = wprefix + incl - (cnt[0] + cnt[1]), local1 = local0 + cnt[0];
    *reinterpret_cast<uint2*>(&s_local[d0]) = make_uint2(local0, local1);
    *reinterpret_cast<uint2*>(&s_global[d0]) = make_uint2(my_base[0] + excl_tiles[0] - local0, my_base[1] + excl_tiles[1] - local1);
    __syncthreads();
    // ---- scatter into the tile's sorted order in shared memory
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
      if (warp_base + r * 32 + lane < n) {
        const unsigned int digit = (key[r] >> shift) & (RADIX - 1);
        const unsigned int pos = s_local[digit] + warp_hist[warp][digit] + rank[r];
        s_keys[pos] = key[r]; s_vals[pos] = val[r];
      }
    }
    __syncthreads();
    // ---- coalesced write-out: consecutive slots of one digit go to consecutive global positions
    const unsigned int valid_n = min((unsigned int)TILE_N, n - tile_base);
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
      const unsigned int slot = r * SORT_THREADS + threadIdx.x;
      if (slot < valid_n) {
        const unsigned int k = s_keys[slot];
        const unsigned int out = s_global[(k >> shift) & (RADIX - 1)] + slot;
        const unsigned int v = s_vals[slot];
        if (MODE != 0 && gather) {
          const ushort4 rc = rect[v];
          ids_out[out] = v; ys_out[out] = (unsigned int)rc.y | ((unsigned int)rc.w << 16); xs_out[out] = (unsigned int)rc.x | ((unsigned int)rc.z << 16);
        } else { keys_out[out] = k; vals_out[out] = v; }
      }
    }
    __syncthreads();
  }
}

void launch_sort_depth(const Workspace& ws, long long max_count, int num_sms, cudaStream_t st) {
  if (max_count <= 0) return;
  const int tile_n = SORT_THREADS * SORT_ITEMS_L1;
  const long long tiles = (max_count + tile_n - 1) / tile_n;
  const int grid = (int)(tiles < 4LL * num_sms ? tiles : 4LL * num_sms);
  int cur = 0;
  for (int p = 0; p < DEPTH_PASSES; ++p) {      // the look-back region of every pass was cleared with the header (fdgs_preprocess)
#define FDGS_PASS(MODEV) onesweep_kernel<SORT_ITEMS_L1, MODEV><<<grid, SORT_THREADS, 0, st>>>(ws.l1_keys[cur], ws.l1_vals[cur], ws.l1_keys[cur ^ 1], ws.l1_vals[cur ^ 1], \
                                                                 &ws.hdr->num_visible, &ws.hdr->sort_ticket[p], ws.sort_hist + p * RADIX, ws.sort_hist + 3 * RADIX,    \
                                                                 reinterpret_cast<unsigned long long*>(ws.sort_lookback + (size_t)p * ws.lookback_stride),             \
                                                                 p * RADIX_BITS, ws.rect, ws.sorted_ys, ws.sorted_xs, ws.sorted_ids)
    if (p == 3) FDGS_PASS(2); else if (p == 2) FDGS_PASS(1); else FDGS_PASS(0);
#undef FDGS_PASS
    count_launch();
    cur ^= 1;
  }
}

}  // namespace fdgs
