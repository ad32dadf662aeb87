// preprocess.cu — K1 (A1-A4 forward) and K8 (B2: backward of A4..A1) for sm_100a.
// One thread per primitive.  The geometry block (68 B/primitive: 4 x float4 + 1 float) is read with
// coalesced 128-bit loads by every thread, because the temporal cull needs it; the colour block
// (12K B/primitive, 89 % of the record at K=48) is read only by survivors.
#include "geom.cuh"

namespace fdgs {

long long g_launches = 0;

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
  ++g_launches;
}

void launch_preprocess_fwd(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, cudaStream_t st) {
  if (sc.N <= 0) return;
  const int threads = 128, blocks = (sc.N + threads - 1) / threads;
  const int KD = (sc.sh_degree + 1) * (sc.sh_degree + 1);
#define FDGS_LAUNCH(KDV) preprocess_fwd_kernel<KDV><<<blocks, threads, 0, st>>>(sc, vp, cp, ws.rec, ws.rect, ws.tiles_touched, ws.tile_diff, ws.aux)
  if (KD == 1) FDGS_LAUNCH(1); else if (KD == 4) FDGS_LAUNCH(4); else if (KD == 9) FDGS_LAUNCH(9); else FDGS_LAUNCH(16);
#undef FDGS_LAUNCH
  ++g_launches;
}

}  // namespace fdgs
