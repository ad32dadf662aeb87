// preprocess.cu — K1 (A1-A4 forward) and K8 (B2: backward of A4..A1) for sm_100a.
// One thread per primitive.  The geometry block (68 B/primitive: 4 x float4 + 1 float) is read with
// coalesced 128-bit loads by every thread, because the temporal cull needs it; the colour block
// (12K B/primitive, 89 % of the record at K=48) is read only by survivors.
#include <atomic>

#include "geom.cuh"

namespace fdgs {

static std::atomic<long long> g_launches{0};
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
long long launch_count_value() { return g_launches.load(std::memory_order_relaxed); }

__device__ __forceinline__ float4 ldg4(const float* p, long long i) { return __ldg(reinterpret_cast<const float4*>(p) + i); }

// 4DSH colour (eq. 20): c_ch = max(0, 0.5 + sum_n cos(2 pi n Delta / T) sum_k coef[n,k,ch] Y_k(dir)).
// Returns the un-clamped value per channel.
template <int KD>
__device__ __forceinline__ void colour_forward(const float* __restrict__ coef, const int n_time, const float dir[3],
                                               const float dt_over_T, float raw[3]) {
  float Y[KD];
  sh_basis<KD>(dir[0], dir[1], dir[2], Y);
  float acc[3] = {0.5f, 0.5f, 0.5f};
  for (int n = 0; n < n_time; ++n) {
    const float cn = cospif(2.0f * (float)n * dt_over_T);
    const float* cf = coef + (size_t)n * KD * 3;
    if constexpr (KD % 4 == 0) {       // 3 x float4 = 4 coefficients x 3 channels; record stride 12K B keeps 16-B alignment
      // all loads of this Fourier order are issued before the first use (volatile asm keeps them together; left alone the
      // compiler recycles four registers and serialises the block into three dependent round trips)
      float4 f[3 * (KD / 4)];
#pragma unroll
      for (int q = 0; q < 3 * (KD / 4); ++q)
        asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(f[q].x), "=f"(f[q].y), "=f"(f[q].z), "=f"(f[q].w)
                     : "l"(reinterpret_cast<const float4*>(cf) + q));
#pragma unroll
      for (int k4 = 0; k4 < KD / 4; ++k4) {
        const float4 f0 = f[3 * k4], f1 = f[3 * k4 + 1], f2 = f[3 * k4 + 2];
        const float y0 = cn * Y[4 * k4], y1 = cn * Y[4 * k4 + 1], y2 = cn * Y[4 * k4 + 2], y3 = cn * Y[4 * k4 + 3];
        acc[0] = fmaf(f0.x, y0, acc[0]); acc[1] = fmaf(f0.y, y0, acc[1]); acc[2] = fmaf(f0.z, y0, acc[2]);
        acc[0] = fmaf(f0.w, y1, acc[0]); acc[1] = fmaf(f1.x, y1, acc[1]); acc[2] = fmaf(f1.y, y1, acc[2]);
        acc[0] = fmaf(f1.z, y2, acc[0]); acc[1] = fmaf(f1.w, y2, acc[1]); acc[2] = fmaf(f2.x, y2, acc[2]);
        acc[0] = fmaf(f2.y, y3, acc[0]); acc[1] = fmaf(f2.z, y3, acc[1]); acc[2] = fmaf(f2.w, y3, acc[2]);
      }
    } else {
#pragma unroll
      for (int k = 0; k < KD; ++k) {
        const float yk = cn * Y[k];
        acc[0] = fmaf(__ldg(cf + 3 * k), yk, acc[0]);
        acc[1] = fmaf(__ldg(cf + 3 * k + 1), yk, acc[1]);
        acc[2] = fmaf(__ldg(cf + 3 * k + 2), yk, acc[2]);
      }
    }
  }
  raw[0] = acc[0]; raw[1] = acc[1]; raw[2] = acc[2];
}

__device__ __forceinline__ void view_dir(const Geom& g, const ViewParams& vp, float dir[3], float& inv_rho) {
  const float dx = g.muc[0] - vp.cam[0], dy = g.muc[1] - vp.cam[1], dz = g.muc[2] - vp.cam[2];
  inv_rho = 1.0f / sqrtf(dx * dx + dy * dy + dz * dz);
  dir[0] = dx * inv_rho; dir[1] = dy * inv_rho; dir[2] = dz * inv_rho;
}

template <int KD>
__global__ void __launch_bounds__(128) preprocess_fwd_kernel(const fdgs_scene sc, const ViewParams vp, const CfgParams cp,
                                                             SplatRec* __restrict__ rec, ushort4* __restrict__ rect,
                                                             unsigned int* __restrict__ tiles_touched,
                                                             int* __restrict__ tile_diff, float4* __restrict__ aux) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  bool visible = false;
  Geom g;
  unsigned int count = 0;
  ushort4 rc = make_ushort4(0, 0, 0, 0);
  float radius = 0.f;
  if (i < sc.N) {
    const int st = geom_forward(ldg4(sc.mean, i), ldg4(sc.log_scale, i), ldg4(sc.quat_l, i), ldg4(sc.quat_r, i),
                                __ldg(sc.opacity_logit + i), vp, cp, g, sc.sh + (size_t)i * sc.n_time * KD * 3, sc.n_time * KD * 12);
    if (st == G_VISIBLE) {
      // support radius and tile rectangle (S9): real-valued r, floor/ceil
      const float mid = 0.5f * (g.a2 + g.c2), hd = 0.5f * (g.a2 - g.c2);
      const float lam = mid + sqrtf(fmaxf(0.f, fmaf(hd, hd, g.b2 * g.b2)));
      radius = cp.cutoff_sigma * sqrtf(lam);
      const float inv = 1.0f / TILE;
      const int tx0 = min(max((int)floorf((g.u - radius) * inv), 0), vp.tiles_x);
      const int ty0 = min(max((int)floorf((g.v - radius) * inv), 0), vp.tiles_y);
      const int tx1 = min(max((int)ceilf((g.u + radius) * inv), 0), vp.tiles_x);
      const int ty1 = min(max((int)ceilf((g.v + radius) * inv), 0), vp.tiles_y);
      if (isfinite(g.u) && isfinite(g.v) && isfinite(radius) && tx1 > tx0 && ty1 > ty0) {
        visible = true;
        count = (unsigned int)(tx1 - tx0) * (unsigned int)(ty1 - ty0);
        rc = make_ushort4(tx0, ty0, tx1, ty1);
      }
    }
    tiles_touched[i] = count;
    rect[i] = rc;
  }
  if (!visible) return;
  {  // coverage count of every tile as a 2D difference array (4 atomics per survivor instead of one per pair);
     // its 2D prefix sum gives the per-tile list lengths, hence the tile ranges and D, before any pair exists
    const int sx = vp.tiles_x + 1;
    atomicAdd(tile_diff + rc.y * sx + rc.x, 1);
    atomicAdd(tile_diff + rc.y * sx + rc.z, -1);
    atomicAdd(tile_diff + rc.w * sx + rc.x, -1);
    atomicAdd(tile_diff + rc.w * sx + rc.z, 1);
  }
  float dir[3], inv_rho, raw[3];
  view_dir(g, vp, dir, inv_rho);
  colour_forward<KD>(sc.sh + (size_t)i * sc.n_time * KD * 3, sc.n_time, dir, g.dt * vp.inv_T, raw);
  aux[i] = make_float4(dir[0], dir[1], dir[2], g.dt * vp.inv_T);     // kept for the colour backward
  // conic = Sigma_2d^-1 = [c2, -b2; -b2, a2] / det, stored as the exp2-scaled Cholesky factor (common.cuh)
  const float kk = 0.72134752044448170f;   // log2(e) / 2
  const float A = g.c2 / g.det, B = -g.b2 / g.det;
  const float ca = sqrtf(kk * A);
  SplatRec r;
  r.u = g.u; r.v = g.v; r.ca = ca; r.cb = kk * B / ca;
  r.cc = sqrtf(kk / g.c2);                  // k (C - B^2/A) = k / c2
  // lo = log2(o), o = sigmoid(logit) * w  (opacity x temporal marginal, eq. 6)
  r.lo = log2f(g.sig) - kk * g.dt * g.dt / g.b;
  r.r = fmaxf(raw[0], 0.f); r.g = fmaxf(raw[1], 0.f); r.b = fmaxf(raw[2], 0.f);
  r.depth = g.p[2]; r.radius = radius; r.w = g.w;
  float4* dst = reinterpret_cast<float4*>(rec + i);
  dst[0] = make_float4(r.u, r.v, r.ca, r.cb);
  dst[1] = make_float4(r.cc, r.lo, r.r, r.g);
  dst[2] = make_float4(r.b, r.depth, r.radius, r.w);
}

// Support radius and tile rectangle of a visible primitive (S9: real-valued r, floor / ceil); count == 0: empty.
__device__ __forceinline__ unsigned int tile_rect(const Geom& g, const ViewParams& vp, const CfgParams& cp, float& radius, ushort4& rc) {
  const float mid = 0.5f * (g.a2 + g.c2), hd = 0.5f * (g.a2 - g.c2);
  const float lam = mid + sqrtf(fmaxf(0.f, fmaf(hd, hd, g.b2 * g.b2)));
  radius = cp.cutoff_sigma * sqrtf(lam);
  const float inv = 1.0f / TILE;
  const int tx0 = min(max((int)floorf((g.u - radius) * inv), 0), vp.tiles_x);
  const int ty0 = min(max((int)floorf((g.v - radius) * inv), 0), vp.tiles_y);
  const int tx1 = min(max((int)ceilf((g.u + radius) * inv), 0), vp.tiles_x);
  const int ty1 = min(max((int)ceilf((g.v + radius) * inv), 0), vp.tiles_y);
  rc = make_ushort4(0, 0, 0, 0);
  if (!(isfinite(g.u) && isfinite(g.v) && isfinite(radius) && tx1 > tx0 && ty1 > ty0)) return 0u;
  rc = make_ushort4(tx0, ty0, tx1, ty1);
  return (unsigned int)(tx1 - tx0) * (unsigned int)(ty1 - ty0);
}

// K1 for sh_degree 3 (KD = 16: every benchmark configuration), in three phases inside a CTA of 128 primitives, so that
// each phase runs on dense warps and every byte of HBM traffic is a byte the method needs:
//   1. one thread per primitive: the 68-byte geometry row, the time row of R, Sigma_44 and the marginal filter (A1 + the
//      temporal half of A2) — three primitives out of four stop here at cfg3, having read 68 bytes; the rest are
//      compacted into a shared list;
//   2. one thread per time-survivor (dense: ~33 of 128): the rest of the chain (slice, projection, conic, radius, tile
//      rectangle: A2-A3), the coverage-grid atomics, and the geometric part of the record handed over in shared memory;
//   3. four lanes per visible survivor: lane l owns the SH orders k = 4l .. 4l+3 of every Fourier order — 48 contiguous
//      bytes per order, so a survivor's 12K-byte colour row is read with 128-bit loads that cover exactly its own
//      sectors (no L2 line prefetch, which over-fetched the mostly culled neighbours: 287 MB read per view for 216 needed
//      in round 1), two shuffle levels join the partial colours, and lanes 0-3 store the 48-byte record and the 16-byte
//      hand-over of the colour backward.
// SPLIT = true (product since late round 2): the kernel stops after phase 2 — the phase-2 thread stores the geometric part
// of the record (colour slots zero) and the colour hand-over (direction, Delta / T) itself, and the colour of the visible
// survivors is evaluated by colour_fwd16_kernel below, which fdgs_render_forward runs on a side stream next to the depth
// sort and the row scatter, i.e. off the critical path of a frame: those are latency-bound launches of a few hundred
// CTAs that leave the memory system idle, and only the blend reads the colour.
constexpr int PF_THREADS = 128;
template <bool SPLIT>
__global__ void __launch_bounds__(PF_THREADS) preprocess_fwd16_kernel(const fdgs_scene sc, const ViewParams vp, const CfgParams cp,
                                                                      SplatRec* __restrict__ rec, ushort4* __restrict__ rect,
                                                                      unsigned int* __restrict__ tiles_touched,
                                                                      int* __restrict__ tile_diff, float4* __restrict__ aux) {
  __shared__ unsigned short s_alive[PF_THREADS];
  __shared__ float4 s_hand[SPLIT ? 1 : PF_THREADS][4];      // per visible survivor: q0 | (cc, lo, depth, radius) | (w, dir x, y, z) | (dt/T, id, -, -)
  __shared__ int s_wcount[PF_THREADS / 32], s_wcount2[PF_THREADS / 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned int lt_mask = (1u << lane) - 1u;
  const int i = blockIdx.x * PF_THREADS + threadIdx.x;
  // ---- phase 1: temporal filter ----
  bool alive = false;
  if (i < sc.N) {
    Geom g; GeomQ q;
    alive = geom_time(ldg4(sc.mean, i), ldg4(sc.log_scale, i), ldg4(sc.quat_l, i), ldg4(sc.quat_r, i), __ldg(sc.opacity_logit + i), vp, cp, g, q) == G_VISIBLE;
    if (!alive) { tiles_touched[i] = 0; rect[i] = make_ushort4(0, 0, 0, 0); }
  }
  const unsigned int bal = __ballot_sync(0xffffffffu, alive);
  if (lane == 0) s_wcount[warp] = __popc(bal);
  __syncthreads();
  int woff = 0, n_alive = 0;
#pragma unroll
  for (int w = 0; w < PF_THREADS / 32; ++w) { if (w < warp) woff += s_wcount[w]; n_alive += s_wcount[w]; }
  if (alive) s_alive[woff + __popc(bal & lt_mask)] = (unsigned short)threadIdx.x;
  __syncthreads();
  // ---- phase 2: the spatial chain on dense warps ----
  bool visible = false;
  float4 h0, h1, h2, h3;
  if ((int)threadIdx.x < n_alive) {
    const int id = blockIdx.x * PF_THREADS + s_alive[threadIdx.x];
    const float4 mean = ldg4(sc.mean, id);
    const float logit = __ldg(sc.opacity_logit + id);
    Geom g;
    const int st = geom_forward(mean, ldg4(sc.log_scale, id), ldg4(sc.quat_l, id), ldg4(sc.quat_r, id), logit, vp, cp, g);
    unsigned int count = 0;
    ushort4 rc = make_ushort4(0, 0, 0, 0);
    float radius = 0.f;
    if (st == G_VISIBLE) count = tile_rect(g, vp, cp, radius, rc);
    tiles_touched[id] = count;
    rect[id] = rc;
    if (count) {
      visible = true;
      const int sx = vp.tiles_x + 1;     // coverage count of every tile as a 2D difference array (4 atomics per survivor)
      atomicAdd(tile_diff + rc.y * sx + rc.x, 1); atomicAdd(tile_diff + rc.y * sx + rc.z, -1);
      atomicAdd(tile_diff + rc.w * sx + rc.x, -1); atomicAdd(tile_diff + rc.w * sx + rc.z, 1);
      float dir[3], inv_rho;
      view_dir(g, vp, dir, inv_rho);
      // conic = Sigma_2d^-1 = [c2, -b2; -b2, a2] / det, stored as the exp2-scaled Cholesky factor (common.cuh)
      const float kk = 0.72134752044448170f;   // log2(e) / 2
      const float A = g.c2 / g.det, B = -g.b2 / g.det;
      const float ca = sqrtf(kk * A);
      h0 = make_float4(g.u, g.v, ca, kk * B / ca);
      h1 = make_float4(sqrtf(kk / g.c2), log2f(g.sig) - kk * g.dt * g.dt / g.b, g.p[2], radius);   // cc = sqrt(k / c2); lo = log2(sigmoid w)
      h2 = make_float4(g.w, dir[0], dir[1], dir[2]);
      h3 = make_float4(g.dt * vp.inv_T, __int_as_float(id), 0.f, 0.f);
      if (SPLIT) {
        float4* dst = reinterpret_cast<float4*>(rec + id);
        dst[0] = h0;                                            // u, v, ca, cb
        dst[1] = make_float4(h1.x, h1.y, 0.f, 0.f);             // cc, lo, (r, g: colour role)
        dst[2] = make_float4(0.f, h1.z, h1.w, h2.x);            // (b), depth, radius, w
        aux[id] = make_float4(h2.y, h2.z, h2.w, h3.x);          // direction and Delta / T: read by the colour role and the colour backward
      }
    }
  }
  if (SPLIT) return;
  const unsigned int bal2 = __ballot_sync(0xffffffffu, visible);
  if (lane == 0) s_wcount2[warp] = __popc(bal2);
  __syncthreads();
  int woff2 = 0, n_vis = 0;
#pragma unroll
  for (int w = 0; w < PF_THREADS / 32; ++w) { if (w < warp) woff2 += s_wcount2[w]; n_vis += s_wcount2[w]; }
  if (visible) { float4* dst = s_hand[woff2 + __popc(bal2 & lt_mask)]; dst[0] = h0; dst[1] = h1; dst[2] = h2; dst[3] = h3; }
  __syncthreads();
  // ---- phase 3: colour, four lanes per survivor ----
  const int l = lane & 3, rec_len = sc.n_time * 48;
  for (int sv = threadIdx.x >> 2; sv < ((n_vis + 7) & ~7); sv += PF_THREADS / 4) {   // whole groups of 8 survivors per warp trip: the shuffles below are warp-wide
    const bool have = sv < n_vis;
    float acc[3] = {0.f, 0.f, 0.f};
    float4 q0 = make_float4(0.f, 0.f, 0.f, 0.f), q1 = q0, q2 = q0, q3 = q0;
    int id = 0;
    if (have) {
      q0 = s_hand[sv][0]; q1 = s_hand[sv][1]; q2 = s_hand[sv][2]; q3 = s_hand[sv][3];
      id = __float_as_int(q3.y);
      float Yf[16], Y[4];
      sh_basis<16>(q2.y, q2.z, q2.w, Yf);
#define FDGS_PICK(L0) { _Pragma("unroll") for (int k = 0; k < 4; ++k) Y[k] = Yf[4 * L0 + k]; }
      if (l == 0) FDGS_PICK(0) else if (l == 1) FDGS_PICK(1) else if (l == 2) FDGS_PICK(2) else FDGS_PICK(3)
#undef FDGS_PICK
      const float4* c4p = reinterpret_cast<const float4*>(sc.sh + (size_t)id * rec_len) + 3 * l;
      for (int n0 = 0; n0 < sc.n_time; n0 += 3) {          // up to three Fourier orders (nine 128-bit loads per lane) in flight
        float4 f[9];
#pragma unroll
        for (int m = 0; m < 3; ++m)
          if (n0 + m < sc.n_time) {
#pragma unroll
            for (int qq = 0; qq < 3; ++qq)
              asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(f[3 * m + qq].x), "=f"(f[3 * m + qq].y), "=f"(f[3 * m + qq].z), "=f"(f[3 * m + qq].w)
                           : "l"(c4p + 12 * (n0 + m) + qq));
          }
#pragma unroll
        for (int m = 0; m < 3; ++m)
          if (n0 + m < sc.n_time) {
            const float cn = cospif(2.0f * (float)(n0 + m) * q3.x);
            const float4 f0 = f[3 * m], f1 = f[3 * m + 1], f2 = f[3 * m + 2];
            const float y0 = cn * Y[0], y1 = cn * Y[1], y2 = cn * Y[2], y3 = cn * Y[3];
            acc[0] = fmaf(f0.x, y0, acc[0]); acc[1] = fmaf(f0.y, y0, acc[1]); acc[2] = fmaf(f0.z, y0, acc[2]);
            acc[0] = fmaf(f0.w, y1, acc[0]); acc[1] = fmaf(f1.x, y1, acc[1]); acc[2] = fmaf(f1.y, y1, acc[2]);
            acc[0] = fmaf(f1.z, y2, acc[0]); acc[1] = fmaf(f1.w, y2, acc[1]); acc[2] = fmaf(f2.x, y2, acc[2]);
            acc[0] = fmaf(f2.y, y3, acc[0]); acc[1] = fmaf(f2.z, y3, acc[1]); acc[2] = fmaf(f2.w, y3, acc[2]);
          }
      }
    }
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
      acc[0] += __shfl_xor_sync(0xffffffffu, acc[0], o); acc[1] += __shfl_xor_sync(0xffffffffu, acc[1], o); acc[2] += __shfl_xor_sync(0xffffffffu, acc[2], o);
    }
    if (have) {
      const float r = fmaxf(acc[0] + 0.5f, 0.f), gch = fmaxf(acc[1] + 0.5f, 0.f), b = fmaxf(acc[2] + 0.5f, 0.f);
      float4* dst = reinterpret_cast<float4*>(rec + id);
      if (l == 0) dst[0] = q0;                                             // u, v, ca, cb
      else if (l == 1) dst[1] = make_float4(q1.x, q1.y, r, gch);           // cc, lo, r, g
      else if (l == 2) dst[2] = make_float4(b, q1.z, q1.w, q2.x);          // b, depth, radius, w
      else aux[id] = make_float4(q2.y, q2.z, q2.w, q3.x);                  // kept for the colour backward
    }
  }
}

// A4 for the visible survivors of a degree-3 scene (eq. 20), after preprocess_fwd16_kernel<true> and the compaction: four
// lanes per survivor (dense: the survivors come from the compacted id list), lane l owns the SH orders 4l .. 4l+3 of every
// Fourier order — 48 contiguous bytes per order, three 128-bit loads — two shuffle levels join the partial sums, and the
// three colour slots of the record are filled in.  The survivor count lives on the device: grid-stride over groups of 8.
constexpr int CF_THREADS = 256;
__global__ void __launch_bounds__(CF_THREADS) colour_fwd16_kernel(const float* __restrict__ sh, const int n_time, const float4* __restrict__ aux,
                                                                  const unsigned int* __restrict__ vis_ids, const WsHeader* __restrict__ hdr,
                                                                  SplatRec* __restrict__ rec) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, l = lane & 3;
  const unsigned int n = hdr->num_visible;
  const int rec_len = n_time * 48;
  constexpr unsigned int PER_CTA = CF_THREADS / 4;
  const unsigned int stride = gridDim.x * PER_CTA;
  // the id and the hand-over of the NEXT group are requested before the coefficient loads of the current one: a trip is one
  // memory round trip instead of three dependent ones (id -> direction -> coefficients)
  unsigned int base = blockIdx.x * PER_CTA + warp * 8;
  unsigned int id_n = 0;
  float4 a_n = make_float4(0.f, 0.f, 0.f, 0.f);
  if (base + (lane >> 2) < n) { id_n = vis_ids[base + (lane >> 2)]; a_n = __ldg(aux + id_n); }
  for (; base < n; base += stride) {     // warp-uniform trip count
    const bool have = base + (lane >> 2) < n;
    const unsigned int id = id_n;
    const float4 a = a_n;
    const float4* c4p = reinterpret_cast<const float4*>(sh + (size_t)id * rec_len) + 3 * l;
    float4 f[9];
    if (have) {
#pragma unroll
      for (int m = 0; m < 3; ++m)
        if (m < n_time) {
#pragma unroll
          for (int qq = 0; qq < 3; ++qq)
            asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(f[3 * m + qq].x), "=f"(f[3 * m + qq].y), "=f"(f[3 * m + qq].z), "=f"(f[3 * m + qq].w)
                         : "l"(c4p + 12 * m + qq));
        }
    }
    const unsigned int sv_n = base + stride + (lane >> 2);
    if (sv_n < n) { id_n = vis_ids[sv_n]; a_n = __ldg(aux + id_n); }
    float acc[3] = {0.f, 0.f, 0.f};
    if (have) {
      float Yf[16], Y[4];
      sh_basis<16>(a.x, a.y, a.z, Yf);
#define FDGS_PICK(L0) { _Pragma("unroll") for (int k = 0; k < 4; ++k) Y[k] = Yf[4 * L0 + k]; }
      if (l == 0) FDGS_PICK(0) else if (l == 1) FDGS_PICK(1) else if (l == 2) FDGS_PICK(2) else FDGS_PICK(3)
#undef FDGS_PICK
      for (int n0 = 0; n0 < n_time; n0 += 3) {          // three Fourier orders (nine 128-bit loads per lane) at a time
        if (n0 > 0) {
#pragma unroll
          for (int m = 0; m < 3; ++m)
            if (n0 + m < n_time) {
#pragma unroll
              for (int qq = 0; qq < 3; ++qq)
                asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(f[3 * m + qq].x), "=f"(f[3 * m + qq].y), "=f"(f[3 * m + qq].z), "=f"(f[3 * m + qq].w)
                             : "l"(c4p + 12 * (n0 + m) + qq));
            }
        }
#pragma unroll
        for (int m = 0; m < 3; ++m)
          if (n0 + m < n_time) {
            const float cn = cospif(2.0f * (float)(n0 + m) * a.w);
            const float4 f0 = f[3 * m], f1 = f[3 * m + 1], f2 = f[3 * m + 2];
            const float y0 = cn * Y[0], y1 = cn * Y[1], y2 = cn * Y[2], y3 = cn * Y[3];
            acc[0] = fmaf(f0.x, y0, acc[0]); acc[1] = fmaf(f0.y, y0, acc[1]); acc[2] = fmaf(f0.z, y0, acc[2]);
            acc[0] = fmaf(f0.w, y1, acc[0]); acc[1] = fmaf(f1.x, y1, acc[1]); acc[2] = fmaf(f1.y, y1, acc[2]);
            acc[0] = fmaf(f1.z, y2, acc[0]); acc[1] = fmaf(f1.w, y2, acc[1]); acc[2] = fmaf(f2.x, y2, acc[2]);
            acc[0] = fmaf(f2.y, y3, acc[0]); acc[1] = fmaf(f2.z, y3, acc[1]); acc[2] = fmaf(f2.w, y3, acc[2]);
          }
      }
    }
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
      acc[0] += __shfl_xor_sync(0xffffffffu, acc[0], o); acc[1] += __shfl_xor_sync(0xffffffffu, acc[1], o); acc[2] += __shfl_xor_sync(0xffffffffu, acc[2], o);
    }
    if (have) {
      float* dst = reinterpret_cast<float*>(rec + id);            // q1 = (cc, lo, r, g), q2 = (b, depth, radius, w)
      if (l == 1) *reinterpret_cast<float2*>(dst + 6) = make_float2(fmaxf(acc[0] + 0.5f, 0.f), fmaxf(acc[1] + 0.5f, 0.f));
      else if (l == 2) dst[8] = fmaxf(acc[2] + 0.5f, 0.f);
    }
  }
}

bool launch_colour_fwd(const fdgs_scene& sc, const Workspace& ws, int num_sms, cudaStream_t st) {
  if (sc.N <= 0 || sc.sh_degree != 3) return false;      // the other degrees evaluate the colour inside preprocess_fwd_kernel<KD>
  const long long groups = ((long long)sc.N + CF_THREADS / 4 - 1) / (CF_THREADS / 4);
    // two CTAs per SM: the kernel shares the GPU with the depth sort, whose passes are chains of ~126 CTAs that slow down when
  // they have to queue for an SM (measured at cfg3, frame ms: 1 per SM 0.503, 2: 0.493, 3: 0.501, 4: 0.506, 16: 0.507)
  const int grid = (int)(groups < 2LL * num_sms ? groups : 2LL * num_sms);
  colour_fwd16_kernel<<<grid, CF_THREADS, 0, st>>>(sc.sh, sc.n_time, ws.aux, ws.vis_ids, ws.hdr, ws.rec);
  count_launch();
  return true;
}

// Parity / measurement hook: the cull decision of every primitive (GeomStatus; 3 = empty tile rectangle), recomputed
// from the parameters with the same device functions as the forward.
__global__ void cull_status_kernel(const fdgs_scene sc, const ViewParams vp, const CfgParams cp, unsigned char* __restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= sc.N) return;
  Geom g;
  int st = geom_forward(ldg4(sc.mean, i), ldg4(sc.log_scale, i), ldg4(sc.quat_l, i), ldg4(sc.quat_r, i), __ldg(sc.opacity_logit + i), vp, cp, g);
  if (st == G_VISIBLE) {
    const float mid = 0.5f * (g.a2 + g.c2), hd = 0.5f * (g.a2 - g.c2);
    const float radius = cp.cutoff_sigma * sqrtf(mid + sqrtf(fmaxf(0.f, fmaf(hd, hd, g.b2 * g.b2))));
    const float inv = 1.0f / TILE;
    const int tx0 = min(max((int)floorf((g.u - radius) * inv), 0), vp.tiles_x), ty0 = min(max((int)floorf((g.v - radius) * inv), 0), vp.tiles_y);
    const int tx1 = min(max((int)ceilf((g.u + radius) * inv), 0), vp.tiles_x), ty1 = min(max((int)ceilf((g.v + radius) * inv), 0), vp.tiles_y);
    if (!(isfinite(g.u) && isfinite(g.v) && isfinite(radius) && tx1 > tx0 && ty1 > ty0)) st = G_CULL_RECT;
  }
  dst[i] = (unsigned char)st;
}

void launch_cull_status(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, unsigned char* dst, cudaStream_t st) {
  if (sc.N <= 0) return;
  cull_status_kernel<<<(sc.N + 127) / 128, 128, 0, st>>>(sc, vp, cp, dst);
  count_launch();
}

void launch_preprocess_fwd(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, cudaStream_t st, bool split_colour) {
  if (sc.N <= 0) return;
  const int threads = 128, blocks = (sc.N + threads - 1) / threads;
  const int KD = (sc.sh_degree + 1) * (sc.sh_degree + 1);
#define FDGS_LAUNCH(KDV) preprocess_fwd_kernel<KDV><<<blocks, threads, 0, st>>>(sc, vp, cp, ws.rec, ws.rect, ws.tiles_touched, ws.tile_diff, ws.aux)
  if (KD == 1) FDGS_LAUNCH(1); else if (KD == 4) FDGS_LAUNCH(4); else if (KD == 9) FDGS_LAUNCH(9);
  else if (split_colour) preprocess_fwd16_kernel<true><<<blocks, PF_THREADS, 0, st>>>(sc, vp, cp, ws.rec, ws.rect, ws.tiles_touched, ws.tile_diff, ws.aux);
  else preprocess_fwd16_kernel<false><<<blocks, PF_THREADS, 0, st>>>(sc, vp, cp, ws.rec, ws.rect, ws.tiles_touched, ws.tile_diff, ws.aux);
#undef FDGS_LAUNCH
  count_launch();
}

}  // namespace fdgs
