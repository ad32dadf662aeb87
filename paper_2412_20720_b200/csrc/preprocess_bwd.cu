// preprocess_bwd.cu — K8 (B2): VJP of A4, A3, A2, A1 for every surviving primitive (sm_100a), as two kernels:
//   colour_bwd_kernel  (A4)       HBM-bound, light in registers, many loads in flight;
//   geom_bwd_kernel    (A3..A1)   register-heavy chain, ~300 B per survivor.
// Nothing but the 9 per-splat gradients of the blend backward, the view direction / time offset kept by the forward
// preprocess (ws.aux) and the hand-over vector ws.dcol is read from the workspace; gradients are accumulated (+=)
// into the caller's arrays.
#include "geom.cuh"

namespace fdgs {

__device__ __forceinline__ void ld_nc_f4(const float4* p, float4& v) {
  asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
}
__device__ __forceinline__ void ld_f4(const float4* p, float4& v) {
  asm volatile("ld.global.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
}
__device__ __forceinline__ float4 ldg4b(const float* p, long long i) { return __ldg(reinterpret_cast<const float4*>(p) + i); }

// Per-k gradient of the real SH basis wrt (x,y,z) (polynomial extension), G[k*3 + c].
template <int KD>
__device__ __forceinline__ void sh_grad_table(const float x, const float y, const float z, float* G) {
#pragma unroll
  for (int i = 0; i < 3 * KD; ++i) G[i] = 0.f;
  if (KD > 1) { G[1 * 3 + 1] = -SH_C1; G[2 * 3 + 2] = SH_C1; G[3 * 3 + 0] = -SH_C1; }
  if (KD > 4) {
    G[4 * 3 + 0] = SH_C2 * y;  G[4 * 3 + 1] = SH_C2 * x;
    G[5 * 3 + 1] = -SH_C2 * z; G[5 * 3 + 2] = -SH_C2 * y;
    G[6 * 3 + 0] = -2.f * SH_C20 * x; G[6 * 3 + 1] = -2.f * SH_C20 * y; G[6 * 3 + 2] = 4.f * SH_C20 * z;
    G[7 * 3 + 0] = -SH_C2 * z; G[7 * 3 + 2] = -SH_C2 * x;
    G[8 * 3 + 0] = 2.f * SH_C22 * x; G[8 * 3 + 1] = -2.f * SH_C22 * y;
  }
  if (KD > 9) {
    const float xx = x * x, yy = y * y, zz = z * z;
    G[9 * 3 + 0] = -SH_C3 * 6.f * x * y;  G[9 * 3 + 1] = -SH_C3 * 3.f * (xx - yy);
    G[10 * 3 + 0] = SH_C4 * y * z;        G[10 * 3 + 1] = SH_C4 * x * z;                      G[10 * 3 + 2] = SH_C4 * x * y;
    G[11 * 3 + 0] = SH_C5 * 2.f * x * y;  G[11 * 3 + 1] = -SH_C5 * (4.f * zz - xx - 3.f * yy); G[11 * 3 + 2] = -SH_C5 * 8.f * y * z;
    G[12 * 3 + 0] = -SH_C6 * 6.f * x * z; G[12 * 3 + 1] = -SH_C6 * 6.f * y * z;               G[12 * 3 + 2] = SH_C6 * (6.f * zz - 3.f * xx - 3.f * yy);
    G[13 * 3 + 0] = -SH_C5 * (4.f * zz - 3.f * xx - yy); G[13 * 3 + 1] = SH_C5 * 2.f * x * y;  G[13 * 3 + 2] = -SH_C5 * 8.f * x * z;
    G[14 * 3 + 0] = SH_C4 * x * z;        G[14 * 3 + 1] = -SH_C4 * y * z;                     G[14 * 3 + 2] = SH_C42 * (xx - yy);
    G[15 * 3 + 0] = -SH_C3 * 3.f * (xx - yy); G[15 * 3 + 1] = SH_C3 * 6.f * x * y;
  }
}

constexpr int CB_WARPS = 4;
// per-survivor table in shared memory: Y[16] | gradY[48] | cos_n[8] | -omega_n sin_n [8] | masked dL/dc [3]; odd stride
constexpr int TAB_Y = 0, TAB_G = 16, TAB_CN = 64, TAB_WS = 72, TAB_GC = 80, TAB_STRIDE = 85;

// One element of the 4DSH coefficient record (eq. 20): its own gradient and its share of dL/d dir, dL/d Delta.
template <int KD>
__device__ __forceinline__ void colour_element(const float* __restrict__ t, const int e, const float coef, float& dcoef,
                                               float& ax, float& ay, float& az, float& ad) {
  const int n = e / (3 * KD), rem = e - n * 3 * KD, k = rem / 3, ch = rem - 3 * k;
  const float yk = t[TAB_Y + k], cn = t[TAB_CN + n], gc = t[TAB_GC + ch];
  dcoef = fmaf(gc * cn, yk, dcoef);
  const float sv = coef * gc, sc_n = sv * cn;
  ad = fmaf(sv * t[TAB_WS + n], yk, ad);
  ax = fmaf(sc_n, t[TAB_G + 3 * k], ax); ay = fmaf(sc_n, t[TAB_G + 3 * k + 1], ay); az = fmaf(sc_n, t[TAB_G + 3 * k + 2], az);
}

// K8a (B2, colour part): VJP of A4.  HBM-bound: per survivor it reads the 12K-byte coefficient block and
// read-modify-writes the 12K-byte gradient block.  A warp owns 32 consecutive survivors; lane s first builds survivor
// s's table (SH basis, its gradient, the Fourier factors, the clamp-masked dL/dc); then groups of 4 lanes walk one
// survivor each (8 survivors in flight per warp, 64 contiguous bytes per group and load instruction, three 128-bit
// loads of coefficients and three of gradients issued before the first use), and a 2-level shuffle gives the
// survivor's dL/d dir and dL/d Delta, handed to the geometry kernel through ws.dcol.
template <int KD>
__global__ void __launch_bounds__(32 * CB_WARPS) colour_bwd_kernel(const float* __restrict__ sh, const int n_time, const float inv_T,
                                                                   const unsigned int* __restrict__ vis_list, const WsHeader* __restrict__ hdr,
                                                                   const float* __restrict__ g9, const SplatRec* __restrict__ rec,
                                                                   const float4* __restrict__ aux, float* __restrict__ dsh,
                                                                   float4* __restrict__ dcol) {
  __shared__ float tab[CB_WARPS][32][TAB_STRIDE];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned int n_vis = hdr->num_visible;
  const unsigned int warp_slot = (blockIdx.x * CB_WARPS + warp) * 32;
  if (warp_slot >= n_vis) return;
  const unsigned int slot = warp_slot + lane;
  const bool have = slot < n_vis;
  int i = 0;
  if (have) {
    i = vis_list[slot];
    if (lane < 8) {  // first batch of 8 survivors: both 12K-byte blocks on their way from HBM while the tables are built
      const size_t off = (size_t)i * (n_time * KD * 3);
      prefetch_l2(sh + off, n_time * KD * 12);
      prefetch_l2(dsh + off, n_time * KD * 12);
    }
    float* my = tab[warp][lane];
    const float4 a = __ldg(aux + i);
    float Y[KD], G[3 * KD];
    sh_basis<KD>(a.x, a.y, a.z, Y);
    sh_grad_table<KD>(a.x, a.y, a.z, G);
#pragma unroll
    for (int k = 0; k < KD; ++k) my[TAB_Y + k] = Y[k];
#pragma unroll
    for (int k = 0; k < 3 * KD; ++k) my[TAB_G + k] = G[k];
    for (int n = 0; n < n_time; ++n) {
      my[TAB_CN + n] = cospif(2.0f * (float)n * a.w);
      my[TAB_WS + n] = -6.283185307179586f * (float)n * inv_T * sinpif(2.0f * (float)n * a.w);
    }
    // the colour clamp at 0 was active iff the stored (clamped) colour is 0: those channels carry no gradient
    const float* gp = g9 + (size_t)9 * i;
    const float4 q1 = __ldg(reinterpret_cast<const float4*>(rec + i) + 1);
    const float cb = __ldg(reinterpret_cast<const float*>(rec + i) + 8);
    my[TAB_GC + 0] = q1.z > 0.f ? gp[6] : 0.f; my[TAB_GC + 1] = q1.w > 0.f ? gp[7] : 0.f; my[TAB_GC + 2] = cb > 0.f ? gp[8] : 0.f;
  }
  __syncwarp();
  const int rec_len = n_time * KD * 3, grp = lane >> 2, l = lane & 3;
#pragma unroll 1
  for (int b = 0; b < 4; ++b) {
    const int s = 8 * b + grp;
    if (have && (lane >> 3) == b + 1) {     // next batch's blocks: requested one batch ahead (deeper would thrash L2)
      const size_t off = (size_t)i * rec_len;
      prefetch_l2(sh + off, 4 * rec_len);
      prefetch_l2(dsh + off, 4 * rec_len);
    }
    const int id = __shfl_sync(0xffffffffu, i, s);
    const bool valid = __shfl_sync(0xffffffffu, (int)have, s) != 0;
    float ax = 0.f, ay = 0.f, az = 0.f, ad = 0.f;
    if (valid) {
      const float* t = tab[warp][s];
      const float* coef = sh + (size_t)id * rec_len;
      float* dcoef = dsh + (size_t)id * rec_len;
      if ((rec_len & 3) == 0) {
        const int nv = rec_len >> 2;
        const float4* c4p = reinterpret_cast<const float4*>(coef);
        float4* d4p = reinterpret_cast<float4*>(dcoef);
        for (int j0 = l; j0 < nv; j0 += 12) {       // three float4 per lane and trip: 6 loads in flight
          float4 c4[3], d4[3];
#pragma unroll
          for (int r = 0; r < 3; ++r) if (j0 + 4 * r < nv) { c4[r] = __ldg(c4p + j0 + 4 * r); d4[r] = d4p[j0 + 4 * r]; }
#pragma unroll
          for (int r = 0; r < 3; ++r) {
            const int j = j0 + 4 * r;
            if (j < nv) {
              colour_element<KD>(t, 4 * j, c4[r].x, d4[r].x, ax, ay, az, ad);
              colour_element<KD>(t, 4 * j + 1, c4[r].y, d4[r].y, ax, ay, az, ad);
              colour_element<KD>(t, 4 * j + 2, c4[r].z, d4[r].z, ax, ay, az, ad);
              colour_element<KD>(t, 4 * j + 3, c4[r].w, d4[r].w, ax, ay, az, ad);
              d4p[j] = d4[r];
            }
          }
        }
      } else {
        for (int e = l; e < rec_len; e += 4) {
          float d = dcoef[e];
          colour_element<KD>(t, e, __ldg(coef + e), d, ax, ay, az, ad);
          dcoef[e] = d;
        }
      }
    }
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
      ax += __shfl_xor_sync(0xffffffffu, ax, o); ay += __shfl_xor_sync(0xffffffffu, ay, o);
      az += __shfl_xor_sync(0xffffffffu, az, o); ad += __shfl_xor_sync(0xffffffffu, ad, o);
    }
    if (valid && l == 0) dcol[id] = make_float4(ax, ay, az, ad);
  }
}

// K8a for sh_degree 3 (KD = 16, every benchmark configuration): no shared-memory table and no index arithmetic.  Lane l of
// the 4 lanes of a survivor owns the SH orders k = 4l .. 4l+3 of every Fourier order n: 12 contiguous floats
// (4 orders x 3 channels = three 128-bit loads) of the coefficient block and of its gradient block per n, with the
// (k, channel) pattern of every register known at compile time; the four Y_k, their gradients and the masked dL/dc
// live in registers.  A warp has 8 survivors in flight, 6 x 128-bit loads per lane and Fourier order.  No L2 prefetch here:
// 128-byte prefetch lines over-fetch the (mostly culled) neighbours of a 576-byte block — measured 0.70 -> 0.62 ms/step without.
__global__ void __launch_bounds__(128) colour_bwd16_kernel(const float* __restrict__ sh, const int n_time, const float inv_T,
                                                           const unsigned int* __restrict__ vis_list, const WsHeader* __restrict__ hdr,
                                                           const float* __restrict__ g9, const SplatRec* __restrict__ rec,
                                                           const float4* __restrict__ aux, float* __restrict__ dsh, float4* __restrict__ dcol) {
  const int lane = threadIdx.x & 31;
  const unsigned int n_vis = hdr->num_visible;
  const unsigned int warp_slot = (blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32;
  if (warp_slot >= n_vis) return;
  const int rec_len = n_time * 48, grp = lane >> 2, l = lane & 3;
#pragma unroll 1
  for (int b = 0; b < 4; ++b) {
    const unsigned int slot = warp_slot + 8 * b + grp;
    const bool valid = slot < n_vis;
    float ax = 0.f, ay = 0.f, az = 0.f, ad = 0.f;
    int id = 0;
    if (valid) {
      id = vis_list[slot];
      const float4 a = __ldg(aux + id);                       // view direction, (t - mu_t) / T
      float Yf[16], Gf[48], Y[4], G[12];
      sh_basis<16>(a.x, a.y, a.z, Yf);
      sh_grad_table<16>(a.x, a.y, a.z, Gf);
#define FDGS_PICK(L0) { _Pragma("unroll") for (int k = 0; k < 4; ++k) { Y[k] = Yf[4 * L0 + k]; G[3 * k] = Gf[12 * L0 + 3 * k]; G[3 * k + 1] = Gf[12 * L0 + 3 * k + 1]; G[3 * k + 2] = Gf[12 * L0 + 3 * k + 2]; } }
      if (l == 0) FDGS_PICK(0) else if (l == 1) FDGS_PICK(1) else if (l == 2) FDGS_PICK(2) else FDGS_PICK(3)
#undef FDGS_PICK
      // the colour clamp at 0 was active iff the stored (clamped) colour is 0: those channels carry no gradient
      const float* gp = g9 + (size_t)9 * id;
      const float4 q1 = __ldg(reinterpret_cast<const float4*>(rec + id) + 1);
      const float cbl = __ldg(reinterpret_cast<const float*>(rec + id) + 8);
      const float gc[3] = {q1.z > 0.f ? gp[6] : 0.f, q1.w > 0.f ? gp[7] : 0.f, cbl > 0.f ? gp[8] : 0.f};
      const float4* c4p = reinterpret_cast<const float4*>(sh + (size_t)id * rec_len) + 3 * l;
      float4* d4p = reinterpret_cast<float4*>(dsh + (size_t)id * rec_len) + 3 * l;
      for (int n = 0; n < n_time; ++n, c4p += 12, d4p += 12) {
        // all six 128-bit loads of this Fourier order are issued before anything else (volatile asm keeps them together:
        // left to itself the compiler interleaves each gradient load with the previous store, three serial round trips)
        float4 c0, c1, c2, d0, d1, d2;
        ld_nc_f4(c4p, c0); ld_nc_f4(c4p + 1, c1); ld_nc_f4(c4p + 2, c2);
        ld_f4(d4p, d0); ld_f4(d4p + 1, d1); ld_f4(d4p + 2, d2);
        const float cn = cospif(2.0f * (float)n * a.w);
        const float wsn = -6.283185307179586f * (float)n * inv_T * sinpif(2.0f * (float)n * a.w);
        const float cv[12] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w, c2.x, c2.y, c2.z, c2.w};
        float dv[12] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w, d2.x, d2.y, d2.z, d2.w};
        const float gcn[3] = {gc[0] * cn, gc[1] * cn, gc[2] * cn};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          float t = 0.f;                                      // sum over channels of coef * masked dL/dc
#pragma unroll
          for (int ch = 0; ch < 3; ++ch) { dv[3 * k + ch] = fmaf(gcn[ch], Y[k], dv[3 * k + ch]); t = fmaf(cv[3 * k + ch], gc[ch], t); }
          ad = fmaf(t * wsn, Y[k], ad);
          const float tc = t * cn;
          ax = fmaf(tc, G[3 * k], ax); ay = fmaf(tc, G[3 * k + 1], ay); az = fmaf(tc, G[3 * k + 2], az);
        }
        d4p[0] = make_float4(dv[0], dv[1], dv[2], dv[3]); d4p[1] = make_float4(dv[4], dv[5], dv[6], dv[7]); d4p[2] = make_float4(dv[8], dv[9], dv[10], dv[11]);
      }
    }
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
      ax += __shfl_xor_sync(0xffffffffu, ax, o); ay += __shfl_xor_sync(0xffffffffu, ay, o);
      az += __shfl_xor_sync(0xffffffffu, az, o); ad += __shfl_xor_sync(0xffffffffu, ad, o);
    }
    if (valid && l == 0) dcol[id] = make_float4(ax, ay, az, ad);
  }
}

// K8a for a BATCH of up to 4 views (fdgs_step_batch, sh_degree 3): the colour backward of all V views of a step in one pass
// over the primitives.  A primitive that survives in several views of the batch (54 % of the (view, survivor) pairs of cfg3
// fall on primitives seen by another view too) has its 12K-byte coefficient block read once and its gradient block
// read-modified-written once, instead of once per view: both stay in registers (NT Fourier orders x 12 floats each per lane)
// while the views that see the primitive are walked.  A warp owns 32 consecutive primitives, finds the members of the
// union by ballot and serves 8 of them per round:
//   phase 1  lane (member g, view l): loads that view's direction / time offset (aux), clamp flags (stored colour > 0) and
//            dL/dc (g9) of the member and writes one table row to shared memory: Y[16], dY/d(x,y,z)[48], masked dL/dc,
//            cos / -omega sin of the Fourier orders — every (member, view) pair costs one lane, all loads of a round are
//            independent;
//   phase 2  the 4 lanes of a member (SH orders 4l .. 4l+3, as in colour_bwd16_kernel) walk the views that see it, reading
//            their quarter of the row; dL/d(dir, dt) of each (member, view) goes to that view's dcol.
struct BatchColourArgs {
  int V;
  float inv_T[4];
  const unsigned int* tiles_touched[4];
  const float4* aux[4];
  const SplatRec* rec[4];
  const float* g9[4];
  float4* dcol[4];
};
constexpr int CU_ROW = 76;      // floats per table row: Y 16 | G 48 | gc 3, pad | cos 4 | -omega sin 4

#define FDGS_SEL4(arr, i) ((i) == 0 ? (arr)[0] : (i) == 1 ? (arr)[1] : (i) == 2 ? (arr)[2] : (arr)[3])

// ZERO: the caller's gradient array was cleared for this step (FDGS_STEP_ZERO_GRADS): nothing to read, the sums are written.
template <int NT, bool ZERO>
__global__ void __launch_bounds__(128) colour_bwd16_union_kernel(const float* __restrict__ sh, const int N, const BatchColourArgs A,
                                                                 float* __restrict__ dsh) {
  __shared__ __align__(16) float tab[4][32][CU_ROW];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, grp = lane >> 2, l = lane & 3;
  const int warp_base = (blockIdx.x * (blockDim.x >> 5) + warp) * 32;
  if (warp_base >= N) return;
  unsigned int seen = 0;                                        // bit v: this lane's primitive survives in view v
  if (warp_base + lane < N) {
#pragma unroll
    for (int v = 0; v < 4; ++v) if (v < A.V) seen |= (__ldg(A.tiles_touched[v] + warp_base + lane) > 0u ? 1u : 0u) << v;
  }
  unsigned int members = __ballot_sync(0xffffffffu, seen != 0u);
  constexpr int rec_len = NT * 48;
#pragma unroll 1
  while (members) {                                             // warp-uniform: 8 members of the union per round
    const unsigned int src = __fns(members, 0, grp + 1);        // lane of the grp-th member, 0xffffffff if there is none
    const bool valid = src != 0xffffffffu;
    const unsigned int seen_src = __shfl_sync(0xffffffffu, seen, valid ? src : 0);
    const unsigned int vm = valid ? seen_src : 0u;        // views that see this member
    const int id = warp_base + (valid ? (int)src : 0);
    float4 c[NT][3], d[NT][3];
    float4* d4p = reinterpret_cast<float4*>(dsh + (size_t)id * rec_len) + 3 * l;
    if (valid) {
      const float4* c4p = reinterpret_cast<const float4*>(sh + (size_t)id * rec_len) + 3 * l;
#pragma unroll
      for (int n = 0; n < NT; ++n) { ld_nc_f4(c4p + 12 * n, c[n][0]); ld_nc_f4(c4p + 12 * n + 1, c[n][1]); ld_nc_f4(c4p + 12 * n + 2, c[n][2]); }
      if (!ZERO) {
#pragma unroll
        for (int n = 0; n < NT; ++n) { ld_f4(d4p + 12 * n, d[n][0]); ld_f4(d4p + 12 * n + 1, d[n][1]); ld_f4(d4p + 12 * n + 2, d[n][2]); }
      }
    }
    if (ZERO) {
#pragma unroll
      for (int n = 0; n < NT; ++n) d[n][0] = d[n][1] = d[n][2] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    // ---- phase 1: lane (grp, l) = (member, view l)
    float* row = tab[warp][lane];
    if ((vm >> l) & 1u) {
      const float4 a = __ldg(FDGS_SEL4(A.aux, l) + id);
      const SplatRec* rp = FDGS_SEL4(A.rec, l) + id;
      const float* gp = FDGS_SEL4(A.g9, l) + (size_t)9 * id;
      const float4 q1 = __ldg(reinterpret_cast<const float4*>(rp) + 1);
      const float cbl = __ldg(reinterpret_cast<const float*>(rp) + 8);
      const float g6 = __ldg(gp + 6), g7 = __ldg(gp + 7), g8 = __ldg(gp + 8);
      const float inv_T = FDGS_SEL4(A.inv_T, l);
      float Yf[16], Gf[48];
      sh_basis<16>(a.x, a.y, a.z, Yf);
      sh_grad_table<16>(a.x, a.y, a.z, Gf);
      float4* r4 = reinterpret_cast<float4*>(row);
#pragma unroll
      for (int k = 0; k < 4; ++k) r4[k] = make_float4(Yf[4 * k], Yf[4 * k + 1], Yf[4 * k + 2], Yf[4 * k + 3]);
#pragma unroll
      for (int k = 0; k < 12; ++k) r4[4 + k] = make_float4(Gf[4 * k], Gf[4 * k + 1], Gf[4 * k + 2], Gf[4 * k + 3]);
      // the colour clamp at 0 was active iff the stored (clamped) colour is 0: those channels carry no gradient
      r4[16] = make_float4(q1.z > 0.f ? g6 : 0.f, q1.w > 0.f ? g7 : 0.f, cbl > 0.f ? g8 : 0.f, 0.f);
      float cn[4] = {0.f, 0.f, 0.f, 0.f}, wsn[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int n = 0; n < NT; ++n) {
        cn[n] = cospif(2.0f * (float)n * a.w);
        wsn[n] = -6.283185307179586f * (float)n * inv_T * sinpif(2.0f * (float)n * a.w);
      }
      r4[17] = make_float4(cn[0], cn[1], cn[2], cn[3]);
      r4[18] = make_float4(wsn[0], wsn[1], wsn[2], wsn[3]);
    }
    __syncwarp();
    // ---- phase 2: the 4 lanes of a member walk the views that see it
    unsigned int rem = vm;
    float4 mine = make_float4(0.f, 0.f, 0.f, 0.f);              // lane l keeps dL/d(dir, dt) of view l
#pragma unroll 1
    while (__any_sync(0xffffffffu, rem != 0u)) {
      const bool act = rem != 0u;
      const int v = act ? __ffs(rem) - 1 : 0;
      rem &= rem - 1;
      float ax = 0.f, ay = 0.f, az = 0.f, ad = 0.f;
      if (act) {
        const float4* r4 = reinterpret_cast<const float4*>(tab[warp][4 * grp + v]);
        const float4 y4 = r4[l], ga = r4[4 + 3 * l], gb = r4[5 + 3 * l], gcv = r4[6 + 3 * l], g4 = r4[16], cn4 = r4[17], ws4 = r4[18];
        const float Y[4] = {y4.x, y4.y, y4.z, y4.w};
        const float G[12] = {ga.x, ga.y, ga.z, ga.w, gb.x, gb.y, gb.z, gb.w, gcv.x, gcv.y, gcv.z, gcv.w};
        const float gc[3] = {g4.x, g4.y, g4.z};
        const float cns[4] = {cn4.x, cn4.y, cn4.z, cn4.w}, wss[4] = {ws4.x, ws4.y, ws4.z, ws4.w};
#pragma unroll
        for (int n = 0; n < NT; ++n) {
          const float cn = cns[n], wsn = wss[n];
          const float cv[12] = {c[n][0].x, c[n][0].y, c[n][0].z, c[n][0].w, c[n][1].x, c[n][1].y, c[n][1].z, c[n][1].w, c[n][2].x, c[n][2].y, c[n][2].z, c[n][2].w};
          float* dv = reinterpret_cast<float*>(&d[n][0]);
          const float gcn[3] = {gc[0] * cn, gc[1] * cn, gc[2] * cn};
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            float t = 0.f;                                      // sum over channels of coef * masked dL/dc
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) { dv[3 * k + ch] = fmaf(gcn[ch], Y[k], dv[3 * k + ch]); t = fmaf(cv[3 * k + ch], gc[ch], t); }
            ad = fmaf(t * wsn, Y[k], ad);
            const float tc = t * cn;
            ax = fmaf(tc, G[3 * k], ax); ay = fmaf(tc, G[3 * k + 1], ay); az = fmaf(tc, G[3 * k + 2], az);
          }
        }
      }
#pragma unroll
      for (int o = 1; o <= 2; o <<= 1) {
        ax += __shfl_xor_sync(0xffffffffu, ax, o); ay += __shfl_xor_sync(0xffffffffu, ay, o);
        az += __shfl_xor_sync(0xffffffffu, az, o); ad += __shfl_xor_sync(0xffffffffu, ad, o);
      }
      if (act && v == l) mine = make_float4(ax, ay, az, ad);
    }
    if ((vm >> l) & 1u) FDGS_SEL4(A.dcol, l)[id] = mine;
    if (valid) {
#pragma unroll
      for (int n = 0; n < NT; ++n) { d4p[12 * n] = d[n][0]; d4p[12 * n + 1] = d[n][1]; d4p[12 * n + 2] = d[n][2]; }
    }
    __syncwarp();                                               // the table is rewritten in the next round
#pragma unroll
    for (int k = 0; k < 8; ++k) members &= members - 1;          // drop the 8 members served (x & (x - 1) of 0 is 0)
  }
}
#undef FDGS_SEL4

// K8b (B2, geometry part): VJP of A3, A2, A1 for every survivor.  Recomputes the forward chain from the raw parameters
// and accumulates (+=) into the caller's gradient arrays.  One thread owns one primitive, so the read-modify-write
// needs no atomics.  The chain is differentiated in the same factor form the forward uses (geom.cuh):
// Sigma_2d = B B^T + dI, B = T N, N = M3 - c m4^T / b, c = M3 m4, b = m4.m4, M = R diag(s), R = L(q_l) R(q_r).
// ATOMIC (the batched step): the views of a batch run this kernel side by side, so the sums go to the caller's arrays as
// vector reductions (red.global.add.v4.f32) instead of a read-modify-write by the owning thread, and nothing is read back.
__device__ __forceinline__ void red_add_f4(float4* p, const float4 v) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
template <bool ATOMIC>
__global__ void __launch_bounds__(128) geom_bwd_kernel(const fdgs_scene sc, const ViewParams vp, const CfgParams cp,
                                                       const unsigned int* __restrict__ vis_list, const WsHeader* __restrict__ hdr,
                                                       const float* __restrict__ g9, const float4* __restrict__ dcol, const float* __restrict__ gz, const fdgs_grads gr) {
  const unsigned int slot = blockIdx.x * blockDim.x + threadIdx.x;
  if (slot >= hdr->num_visible) return;
  const int i = vis_list[slot];
  Geom g;
  {
    const float4 mean = ldg4b(sc.mean, i), ls = ldg4b(sc.log_scale, i), qlr = ldg4b(sc.quat_l, i), qrr = ldg4b(sc.quat_r, i);
    if (geom_forward(mean, ls, qlr, qrr, __ldg(sc.opacity_logit + i), vp, cp, g) != G_VISIBLE) return;
  }
  // the gradient rows this thread will read-modify-write: requested now, consumed at the end of the chain (the compiler
  // would otherwise issue each load right before its use: five serial round trips on a 12-warps-per-SM kernel)
  float4 acc_mean = make_float4(0.f, 0.f, 0.f, 0.f), acc_ls = acc_mean, acc_ql = acc_mean, acc_qr = acc_mean;
  float acc_logit = 0.f;
  if (!ATOMIC) {
    ld_f4(reinterpret_cast<const float4*>(gr.mean) + i, acc_mean);
    ld_f4(reinterpret_cast<const float4*>(gr.log_scale) + i, acc_ls);
    ld_f4(reinterpret_cast<const float4*>(gr.quat_l) + i, acc_ql);
    ld_f4(reinterpret_cast<const float4*>(gr.quat_r) + i, acc_qr);
    acc_logit = gr.opacity_logit[i];
  }
  const float* gp = g9 + (size_t)9 * i;
  const float g_u = gp[0], g_v = gp[1], g_A = gp[2], g_B = gp[3], g_C = gp[4], g_o = gp[5];
  if (gr.mean2d) {
    if (ATOMIC) { atomicAdd(gr.mean2d + 2 * i, g_u); atomicAdd(gr.mean2d + 2 * i + 1, g_v); }
    else { gr.mean2d[2 * i] += g_u; gr.mean2d[2 * i + 1] += g_v; }
  }
  float dir[3], inv_rho;
  {
    const float dx = g.muc[0] - vp.cam[0], dy = g.muc[1] - vp.cam[1], dz = g.muc[2] - vp.cam[2];
    inv_rho = 1.0f / sqrtf(dx * dx + dy * dy + dz * dz);
    dir[0] = dx * inv_rho; dir[1] = dy * inv_rho; dir[2] = dz * inv_rho;
  }
  const float4 dc = __ldg(dcol + i);
  const float gdx = dc.x, gdy = dc.y, gdz = dc.z, e_dt = dc.w;
  float d_muc[3] = {0.f, 0.f, 0.f}, d_dt = e_dt, d_b = 0.f;
  {
    const float dd = gdx * dir[0] + gdy * dir[1] + gdz * dir[2];
    d_muc[0] = (gdx - dir[0] * dd) * inv_rho; d_muc[1] = (gdy - dir[1] * dd) * inv_rho; d_muc[2] = (gdz - dir[2] * dd) * inv_rho;
  }

  // ---- conic -> Sigma_2d -> B -> (T, N) ------------------------------------------------------
  // G2 = -Q G_Q Q with G_Q = [[g_A, g_B/2],[g_B/2, g_C]], dB = 2 G2 B, dT = dB N^T, dN = T^T dB.
  // For elongated splats Q is nearly singular and these products cancel by the squared axis ratio, so this block
  // (about 100 DFMA per survivor) is carried in fp64 from the fp32 factor B.
  float dT[2][3], dNm[3][4];
  {
    double Bd[2][4], n0 = 0.0, n1 = 0.0, d01 = 0.0, minors = 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) { Bd[0][k] = g.Bm[0][k]; Bd[1][k] = g.Bm[1][k]; n0 = fma(Bd[0][k], Bd[0][k], n0); n1 = fma(Bd[1][k], Bd[1][k], n1); d01 = fma(Bd[0][k], Bd[1][k], d01); }
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
      for (int q = p + 1; q < 4; ++q) { const double m = Bd[0][p] * Bd[1][q] - Bd[0][q] * Bd[1][p]; minors = fma(m, m, minors); }
    const double dil = cp.dilation, det = fma(dil, dil + n0 + n1, minors), idet = 1.0 / det;
    const double A = (n1 + dil) * idet, B = -d01 * idet, C = (n0 + dil) * idet;
    const double h = 0.5 * (double)g_B, gA = g_A, gC = g_C;
    const double qg00 = A * gA + B * h, qg01 = A * h + B * gC, qg10 = B * gA + C * h, qg11 = B * h + C * gC;
    const double G2_00 = -(qg00 * A + qg01 * B), G2_01 = -(qg00 * B + qg01 * C), G2_11 = -(qg10 * B + qg11 * C);
    double dB[2][4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      dB[0][k] = 2.0 * (G2_00 * Bd[0][k] + G2_01 * Bd[1][k]);
      dB[1][k] = 2.0 * (G2_01 * Bd[0][k] + G2_11 * Bd[1][k]);
    }
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
      for (int q = 0; q < 3; ++q)
        dT[r][q] = (float)(dB[r][0] * g.Nm[q][0] + dB[r][1] * g.Nm[q][1] + dB[r][2] * g.Nm[q][2] + dB[r][3] * g.Nm[q][3]);
#pragma unroll
    for (int q = 0; q < 3; ++q)
#pragma unroll
      for (int k = 0; k < 4; ++k) dNm[q][k] = (float)(g.T[0][q] * dB[0][k] + g.T[1][q] * dB[1][k]);
  }

  // ---- T = J W, J(p), pinhole --------------------------------------------------------------
  {
    const float x = g.p[0], y = g.p[1], z = g.p[2], iz = 1.0f / z, iz2 = iz * iz;
    float dJ00 = 0.f, dJ02 = 0.f, dJ11 = 0.f, dJ12 = 0.f;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      dJ00 = fmaf(dT[0][q], vp.W[0][q], dJ00); dJ02 = fmaf(dT[0][q], vp.W[2][q], dJ02);
      dJ11 = fmaf(dT[1][q], vp.W[1][q], dJ11); dJ12 = fmaf(dT[1][q], vp.W[2][q], dJ12);
    }
    float dp[3];
    dp[0] = g_u * vp.fx * iz;
    dp[1] = g_v * vp.fy * iz;
    dp[2] = -(g_u * vp.fx * x + g_v * vp.fy * y) * iz2 - (dJ00 * vp.fx + dJ11 * vp.fy) * iz2;
    if (gz) dp[2] += gz[i];                       // auxiliary depth channel: z_k = p_z
    if (!g.clampx) { dp[0] -= dJ02 * vp.fx * iz2; dp[2] += dJ02 * 2.f * vp.fx * x * iz2 * iz; }
    else           { dp[2] += dJ02 * vp.fx * g.xr * iz2; }
    if (!g.clampy) { dp[1] -= dJ12 * vp.fy * iz2; dp[2] += dJ12 * 2.f * vp.fy * y * iz2 * iz; }
    else           { dp[2] += dJ12 * vp.fy * g.yr * iz2; }
#pragma unroll
    for (int r = 0; r < 3; ++r) d_muc[r] += vp.W[0][r] * dp[0] + vp.W[1][r] * dp[1] + vp.W[2][r] * dp[2];
  }

  // ---- o = sigmoid(logit) w,  w = exp(-Delta^2 / 2b) -----------------------------------------
  const float inv_b = 1.0f / g.b;
  if (ATOMIC) atomicAdd(gr.opacity_logit + i, g_o * g.w * g.sig * g.sig_neg);
  else gr.opacity_logit[i] = acc_logit + g_o * g.w * g.sig * g.sig_neg;
  {
    const float d_w = g_o * g.sig;
    d_dt += d_w * g.w * (-g.dt * inv_b);
    d_b += d_w * g.w * (0.5f * g.dt * g.dt * inv_b * inv_b);
  }
  // ---- mu_c = mu_1:3 + c Delta / b -----------------------------------------------------------
  float d_c[3];
  {
    const float mc = d_muc[0] * g.c[0] + d_muc[1] * g.c[1] + d_muc[2] * g.c[2];
#pragma unroll
    for (int r = 0; r < 3; ++r) d_c[r] = d_muc[r] * g.dt * inv_b;
    d_dt += mc * inv_b;
    d_b += -mc * g.dt * inv_b * inv_b;
  }
  // ---- N = M3 - c m4^T / b;  c = M3 m4;  b = m4.m4 -------------------------------------------
  float dM[4][4];
  {
    float hv[3], ch = 0.f;
#pragma unroll
    for (int r = 0; r < 3; ++r) {
      hv[r] = dNm[r][0] * g.M[3][0] + dNm[r][1] * g.M[3][1] + dNm[r][2] * g.M[3][2] + dNm[r][3] * g.M[3][3];
      d_c[r] -= hv[r] * inv_b;
      ch += g.c[r] * hv[r];
    }
    d_b += ch * inv_b * inv_b;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      float dm4 = -(g.c[0] * dNm[0][k] + g.c[1] * dNm[1][k] + g.c[2] * dNm[2][k]) * inv_b;
      dm4 += d_c[0] * g.M[0][k] + d_c[1] * g.M[1][k] + d_c[2] * g.M[2][k];
      dm4 += 2.f * d_b * g.M[3][k];
      dM[3][k] = dm4;
#pragma unroll
      for (int r = 0; r < 3; ++r) dM[r][k] = dNm[r][k] + d_c[r] * g.M[3][k];
    }
  }
  // ---- mean ---------------------------------------------------------------------------------
  {
    float4* dst = reinterpret_cast<float4*>(gr.mean) + i;
    float4 m = acc_mean;
    m.x += d_muc[0]; m.y += d_muc[1]; m.z += d_muc[2]; m.w += -d_dt;
    if (gr.densify) {   // density-control indicators of this view
      float* dn = gr.densify + (size_t)3 * i;
      if (ATOMIC) { atomicAdd(dn, sqrtf(g_u * g_u + g_v * g_v)); atomicAdd(dn + 1, fabsf(d_dt)); atomicAdd(dn + 2, 1.0f); }
      else { dn[0] += sqrtf(g_u * g_u + g_v * g_v); dn[1] += fabsf(d_dt); dn[2] += 1.0f; }
    }
    if (ATOMIC) red_add_f4(dst, m); else *dst = m;
  }
  // ---- M = R4 diag(s) ------------------------------------------------------------------------
  float dR4[4][4];
  {
    float dls[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      float ds = 0.f;
#pragma unroll
      for (int r = 0; r < 4; ++r) { ds = fmaf(dM[r][k], g.R4[r][k], ds); dR4[r][k] = dM[r][k] * g.s[k]; }
      dls[k] = ds * g.s[k];
    }
    float4* dst = reinterpret_cast<float4*>(gr.log_scale) + i;
    float4 m = acc_ls;
    m.x += dls[0]; m.y += dls[1]; m.z += dls[2]; m.w += dls[3];
    if (ATOMIC) red_add_f4(dst, m); else *dst = m;
  }
  // ---- R4 = L(q_l) R(q_r), quaternion entries, normalisation -----------------------------------
  {
    float Lm[4][4], Rm[4][4], dL[4][4], dR[4][4];
    quat_left(g.ql, Lm); quat_right(g.qr, Rm);
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        dL[r][q] = dR4[r][0] * Rm[q][0] + dR4[r][1] * Rm[q][1] + dR4[r][2] * Rm[q][2] + dR4[r][3] * Rm[q][3];
        dR[r][q] = Lm[0][r] * dR4[0][q] + Lm[1][r] * dR4[1][q] + Lm[2][r] * dR4[2][q] + Lm[3][r] * dR4[3][q];
      }
    float dql[4], dqr[4];
    dql[0] = dL[0][0] + dL[1][1] + dL[2][2] + dL[3][3];
    dql[1] = -dL[0][1] + dL[1][0] - dL[2][3] + dL[3][2];
    dql[2] = -dL[0][2] + dL[1][3] + dL[2][0] - dL[3][1];
    dql[3] = -dL[0][3] - dL[1][2] + dL[2][1] + dL[3][0];
    dqr[0] = dR[0][0] + dR[1][1] + dR[2][2] + dR[3][3];
    dqr[1] = -dR[0][1] + dR[1][0] + dR[2][3] - dR[3][2];
    dqr[2] = -dR[0][2] - dR[1][3] + dR[2][0] + dR[3][1];
    dqr[3] = -dR[0][3] + dR[1][2] - dR[2][1] + dR[3][0];
    float dl = 0.f, dr = 0.f;
#pragma unroll
    for (int k = 0; k < 4; ++k) { dl = fmaf(g.ql[k], dql[k], dl); dr = fmaf(g.qr[k], dqr[k], dr); }
    float4* dstl = reinterpret_cast<float4*>(gr.quat_l) + i;
    float4* dstr = reinterpret_cast<float4*>(gr.quat_r) + i;
    float4 ml = acc_ql, mr = acc_qr;
    ml.x += (dql[0] - g.ql[0] * dl) * g.inv_nl; ml.y += (dql[1] - g.ql[1] * dl) * g.inv_nl;
    ml.z += (dql[2] - g.ql[2] * dl) * g.inv_nl; ml.w += (dql[3] - g.ql[3] * dl) * g.inv_nl;
    mr.x += (dqr[0] - g.qr[0] * dr) * g.inv_nr; mr.y += (dqr[1] - g.qr[1] * dr) * g.inv_nr;
    mr.z += (dqr[2] - g.qr[2] * dr) * g.inv_nr; mr.w += (dqr[3] - g.qr[3] * dr) * g.inv_nr;
    if (ATOMIC) { red_add_f4(dstl, ml); red_add_f4(dstr, mr); } else { *dstl = ml; *dstr = mr; }
  }
}

void launch_preprocess_bwd(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, int l1_buf,
                           const fdgs_grads& gr, bool with_gz, cudaStream_t st) {
  if (sc.N <= 0) return;
  // the survivor count lives on the device: launch for all N slots, surplus warps / threads exit at once
  (void)l1_buf;
  const int KD = (sc.sh_degree + 1) * (sc.sh_degree + 1);
  {
    const int threads = 32 * CB_WARPS, blocks = (sc.N + threads - 1) / threads;
#define FDGS_LAUNCH(KDV) colour_bwd_kernel<KDV><<<blocks, threads, 0, st>>>(sc.sh, sc.n_time, vp.inv_T, ws.vis_ids, ws.hdr, ws.g9, ws.rec, ws.aux, gr.sh, ws.dcol)
    if (KD == 1) FDGS_LAUNCH(1); else if (KD == 4) FDGS_LAUNCH(4); else if (KD == 9) FDGS_LAUNCH(9);
    else colour_bwd16_kernel<<<blocks, threads, 0, st>>>(sc.sh, sc.n_time, vp.inv_T, ws.vis_ids, ws.hdr, ws.g9, ws.rec, ws.aux, gr.sh, ws.dcol);
#undef FDGS_LAUNCH
  }
  geom_bwd_kernel<false><<<(sc.N + 127) / 128, 128, 0, st>>>(sc, vp, cp, ws.vis_ids, ws.hdr, ws.g9, ws.dcol, with_gz ? ws.gz : nullptr, gr);
  count_launch(2);
}

// geometry part alone (the batched step runs it after the batched colour pass, the views side by side: sums by reductions)
void launch_geom_bwd(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, const fdgs_grads& gr, cudaStream_t st) {
  if (sc.N <= 0) return;
  geom_bwd_kernel<true><<<(sc.N + 127) / 128, 128, 0, st>>>(sc, vp, cp, ws.vis_ids, ws.hdr, ws.g9, ws.dcol, nullptr, gr);
  count_launch();
}

// colour part of all V views of a batch in one pass (see colour_bwd16_union_kernel); false = not available for this
// scene (sh_degree != 3 or more than 4 Fourier orders): the caller then runs the per-view kernels
bool launch_colour_bwd_batch(const fdgs_scene& sc, int V, const Workspace* ws, const float* inv_T, const fdgs_grads& gr, bool grads_are_zero,
                             cudaStream_t st) {
  if (sc.sh_degree != 3 || sc.n_time > 4 || V < 1 || V > 4) return false;
  if (sc.N <= 0) return true;
  BatchColourArgs A{};
  A.V = V;
  for (int v = 0; v < V; ++v) {
    A.inv_T[v] = inv_T[v]; A.tiles_touched[v] = ws[v].tiles_touched; A.aux[v] = ws[v].aux; A.rec[v] = ws[v].rec; A.g9[v] = ws[v].g9; A.dcol[v] = ws[v].dcol;
  }
  const int blocks = (sc.N + 127) / 128;
#define FDGS_CU(NTV) do { if (grads_are_zero) colour_bwd16_union_kernel<NTV, true><<<blocks, 128, 0, st>>>(sc.sh, sc.N, A, gr.sh); \
                         else colour_bwd16_union_kernel<NTV, false><<<blocks, 128, 0, st>>>(sc.sh, sc.N, A, gr.sh); } while (0)
  switch (sc.n_time) {
    case 1: FDGS_CU(1); break;
    case 2: FDGS_CU(2); break;
    case 3: FDGS_CU(3); break;
    default: FDGS_CU(4); break;
  }
#undef FDGS_CU
  count_launch();
  return true;
}

}  // namespace fdgs
