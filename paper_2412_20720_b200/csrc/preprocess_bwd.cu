// preprocess_bwd.cu — K8 (B2): VJP of A4, A3, A2, A1 for every surviving primitive (sm_100a).
// Recomputes the forward chain from the raw parameters (nothing but the 9 per-splat gradients of the
// blend backward is read from the workspace) and accumulates (+=) into the caller's gradient arrays.
// One thread owns one primitive, so the read-modify-write needs no atomics.
// The chain is differentiated in the same factor form the forward uses (geom.cuh): Sigma_2d = B B^T + dI,
// B = T N, N = M3 - c m4^T / b, c = M3 m4, b = m4.m4, M = R diag(s), R = L(q_l) R(q_r).
#include "geom.cuh"

namespace fdgs {

__device__ __forceinline__ float4 ldg4b(const float* p, long long i) { return __ldg(reinterpret_cast<const float4*>(p) + i); }

template <int KD>
__global__ void __launch_bounds__(128) preprocess_bwd_kernel(const fdgs_scene sc, const ViewParams vp, const CfgParams cp,
                                                             const unsigned int* __restrict__ vis_list,
                                                             const WsHeader* __restrict__ hdr, const float* __restrict__ g9,
                                                             const fdgs_grads gr) {
  const unsigned int slot = blockIdx.x * blockDim.x + threadIdx.x;
  if (slot >= hdr->num_visible) return;
  const int i = vis_list[slot];
  const float4 mean = ldg4b(sc.mean, i), ls = ldg4b(sc.log_scale, i), qlr = ldg4b(sc.quat_l, i), qrr = ldg4b(sc.quat_r, i);
  const float logit = __ldg(sc.opacity_logit + i);
  Geom g;
  if (geom_forward(mean, ls, qlr, qrr, logit, vp, cp, g) != G_VISIBLE) return;
  const float* gp = g9 + (size_t)9 * i;
  const float g_u = gp[0], g_v = gp[1], g_A = gp[2], g_B = gp[3], g_C = gp[4], g_o = gp[5];
  const float g_c[3] = {gp[6], gp[7], gp[8]};
  if (gr.mean2d) { gr.mean2d[2 * i] += g_u; gr.mean2d[2 * i + 1] += g_v; }
  float d_muc[3] = {0.f, 0.f, 0.f}, d_dt = 0.f, d_b = 0.f;

  // ---- (A4) colour -------------------------------------------------------------------------
  {
    float dir[3], inv_rho;
    {
      const float dx = g.muc[0] - vp.cam[0], dy = g.muc[1] - vp.cam[1], dz = g.muc[2] - vp.cam[2];
      inv_rho = 1.0f / sqrtf(dx * dx + dy * dy + dz * dz);
      dir[0] = dx * inv_rho; dir[1] = dy * inv_rho; dir[2] = dz * inv_rho;
    }
    float Y[KD], a[KD];
    sh_basis<KD>(dir[0], dir[1], dir[2], Y);
#pragma unroll
    for (int k = 0; k < KD; ++k) a[k] = 0.f;
    const float* coef = sc.sh + (size_t)i * sc.n_time * KD * 3;
    float* dcoef = gr.sh + (size_t)i * sc.n_time * KD * 3;
    const float dtT = g.dt * vp.inv_T;
    // first pass: un-clamped colour (the clamp state decides which channels carry gradient)
    float raw[3] = {0.5f, 0.5f, 0.5f};
    for (int n = 0; n < sc.n_time; ++n) {
      const float cn = cospif(2.0f * (float)n * dtT);
      const float* cf = coef + (size_t)n * KD * 3;
#pragma unroll
      for (int k = 0; k < KD; ++k) {
        const float yk = cn * Y[k];
        raw[0] = fmaf(__ldg(cf + 3 * k), yk, raw[0]); raw[1] = fmaf(__ldg(cf + 3 * k + 1), yk, raw[1]); raw[2] = fmaf(__ldg(cf + 3 * k + 2), yk, raw[2]);
      }
    }
    const float gc0 = raw[0] > 0.f ? g_c[0] : 0.f, gc1 = raw[1] > 0.f ? g_c[1] : 0.f, gc2 = raw[2] > 0.f ? g_c[2] : 0.f;
    float e_dt = 0.f;
    for (int n = 0; n < sc.n_time; ++n) {
      const float cn = cospif(2.0f * (float)n * dtT), sn = sinpif(2.0f * (float)n * dtT);
      const float om = 6.283185307179586f * (float)n * vp.inv_T;
      const float* cf = coef + (size_t)n * KD * 3;
      float* dcf = dcoef + (size_t)n * KD * 3;
#pragma unroll
      for (int k = 0; k < KD; ++k) {
        const float yk = cn * Y[k];
        const float s = gc0 * __ldg(cf + 3 * k) + gc1 * __ldg(cf + 3 * k + 1) + gc2 * __ldg(cf + 3 * k + 2);
        dcf[3 * k] += gc0 * yk; dcf[3 * k + 1] += gc1 * yk; dcf[3 * k + 2] += gc2 * yk;
        a[k] = fmaf(cn, s, a[k]);
        e_dt = fmaf(-om * sn * Y[k], s, e_dt);
      }
    }
    d_dt += e_dt;
    float gd[3];
    sh_grad<KD>(dir[0], dir[1], dir[2], a, gd);
    const float dd = gd[0] * dir[0] + gd[1] * dir[1] + gd[2] * dir[2];
#pragma unroll
    for (int r = 0; r < 3; ++r) d_muc[r] += (gd[r] - dir[r] * dd) * inv_rho;
  }

  // ---- conic -> Sigma_2d -> B -> (T, N) ------------------------------------------------------
  const float idet = 1.0f / g.det;
  const float A = g.c2 * idet, B = -g.b2 * idet, C = g.a2 * idet;
  // G2 = -Q G_Q Q,  G_Q = [[g_A, g_B/2],[g_B/2, g_C]]
  const float h = 0.5f * g_B;
  const float qg00 = A * g_A + B * h, qg01 = A * h + B * g_C, qg10 = B * g_A + C * h, qg11 = B * h + C * g_C;
  const float G2_00 = -(qg00 * A + qg01 * B), G2_01 = -(qg00 * B + qg01 * C), G2_11 = -(qg10 * B + qg11 * C);
  float dBm[2][4], dT[2][3], dNm[3][4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    dBm[0][k] = 2.f * (G2_00 * g.Bm[0][k] + G2_01 * g.Bm[1][k]);
    dBm[1][k] = 2.f * (G2_01 * g.Bm[0][k] + G2_11 * g.Bm[1][k]);
  }
#pragma unroll
  for (int r = 0; r < 2; ++r)
#pragma unroll
    for (int q = 0; q < 3; ++q)
      dT[r][q] = dBm[r][0] * g.Nm[q][0] + dBm[r][1] * g.Nm[q][1] + dBm[r][2] * g.Nm[q][2] + dBm[r][3] * g.Nm[q][3];
#pragma unroll
  for (int q = 0; q < 3; ++q)
#pragma unroll
    for (int k = 0; k < 4; ++k) dNm[q][k] = g.T[0][q] * dBm[0][k] + g.T[1][q] * dBm[1][k];

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
    if (!g.clampx) { dp[0] -= dJ02 * vp.fx * iz2; dp[2] += dJ02 * 2.f * vp.fx * x * iz2 * iz; }
    else           { dp[2] += dJ02 * vp.fx * g.xr * iz2; }
    if (!g.clampy) { dp[1] -= dJ12 * vp.fy * iz2; dp[2] += dJ12 * 2.f * vp.fy * y * iz2 * iz; }
    else           { dp[2] += dJ12 * vp.fy * g.yr * iz2; }
#pragma unroll
    for (int r = 0; r < 3; ++r) d_muc[r] += vp.W[0][r] * dp[0] + vp.W[1][r] * dp[1] + vp.W[2][r] * dp[2];
  }

  // ---- o = sigmoid(logit) w,  w = exp(-Delta^2 / 2b) -----------------------------------------
  const float inv_b = 1.0f / g.b;
  gr.opacity_logit[i] += g_o * g.w * g.sig * (1.f - g.sig);
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
    float4 m = *dst;
    m.x += d_muc[0]; m.y += d_muc[1]; m.z += d_muc[2]; m.w += -d_dt;
    *dst = m;
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
    float4 m = *dst;
    m.x += dls[0]; m.y += dls[1]; m.z += dls[2]; m.w += dls[3];
    *dst = m;
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
    float4 ml = *dstl, mr = *dstr;
    ml.x += (dql[0] - g.ql[0] * dl) * g.inv_nl; ml.y += (dql[1] - g.ql[1] * dl) * g.inv_nl;
    ml.z += (dql[2] - g.ql[2] * dl) * g.inv_nl; ml.w += (dql[3] - g.ql[3] * dl) * g.inv_nl;
    mr.x += (dqr[0] - g.qr[0] * dr) * g.inv_nr; mr.y += (dqr[1] - g.qr[1] * dr) * g.inv_nr;
    mr.z += (dqr[2] - g.qr[2] * dr) * g.inv_nr; mr.w += (dqr[3] - g.qr[3] * dr) * g.inv_nr;
    *dstl = ml; *dstr = mr;
  }
}

void launch_preprocess_bwd(const fdgs_scene& sc, const ViewParams& vp, const CfgParams& cp, const Workspace& ws, int l1_buf,
                           const fdgs_grads& gr, cudaStream_t st) {
  if (sc.N <= 0) return;
  // the survivor count lives on the device: launch for all N slots, surplus threads exit at once
  const int threads = 128, blocks = (sc.N + threads - 1) / threads;
  const int KD = (sc.sh_degree + 1) * (sc.sh_degree + 1);
#define FDGS_LAUNCH(KDV) preprocess_bwd_kernel<KDV><<<blocks, threads, 0, st>>>(sc, vp, cp, ws.l1_vals[l1_buf], ws.hdr, ws.g9, gr)
  if (KD == 1) FDGS_LAUNCH(1); else if (KD == 4) FDGS_LAUNCH(4); else if (KD == 9) FDGS_LAUNCH(9); else FDGS_LAUNCH(16);
#undef FDGS_LAUNCH
  ++g_launches;
}

}  // namespace fdgs
