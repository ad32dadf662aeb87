// geom.cuh — per-primitive chain A1-A3 on the device (fp32), shared by the forward and backward
// preprocess kernels.  PAPER.md eq. 7-10 (L126-L145) and eq. 3-4 (L95-L104).
//
// Numerics: eq. 9's Schur complement is NOT evaluated literally — in fp32
// it cancels catastrophically when the temporal axis is tilted into space.  With M = R diag(s)
// (Sigma = M M^T), m4 = last row of M and M3 = first three rows,
//     Sigma_44 = m4.m4,  Sigma_1:3,4 = M3 m4 =: c,  N = M3 - c m4^T / Sigma_44  =>  Sigma_xyz|t = N N^T
// and Sigma_2d = (T N)(T N)^T + dilation I with T = J W; its determinant is taken by Cauchy-Binet as a
// sum of squares.  Algebraically identical to eq. 9 / eq. 4, no subtraction of close numbers.
#pragma once
#include "common.cuh"

namespace fdgs {

struct Geom {
  float s[4], ql[4], qr[4], inv_nl, inv_nr;
  float R4[4][4], M[4][4];
  float dt, b, w;          // Delta = t - mu_t, Sigma_44, marginal weight
  float c[3], muc[3];      // Sigma_1:3,4 and the conditional mean
  float Nm[3][4];
  float p[3], u, v;
  float xr, yr; bool clampx, clampy;
  float T[2][3], Bm[2][4];
  float a2, b2, c2, det;   // Sigma_2d entries (with dilation) and determinant
  float sig, sig_neg;      // sigmoid(logit), sigmoid(-logit) = 1 - sigmoid(logit) without the cancellation
};

enum GeomStatus { G_VISIBLE = 0, G_CULL_TIME = 1, G_CULL_NEAR = 2, G_CULL_RECT = 3, G_CULL_NONFINITE = 4 };

__device__ __forceinline__ void quat_left(const float q[4], float L[4][4]) {
  const float a = q[0], b = q[1], c = q[2], d = q[3];
  L[0][0] = a; L[0][1] = -b; L[0][2] = -c; L[0][3] = -d;
  L[1][0] = b; L[1][1] = a;  L[1][2] = -d; L[1][3] = c;
  L[2][0] = c; L[2][1] = d;  L[2][2] = a;  L[2][3] = -b;
  L[3][0] = d; L[3][1] = -c; L[3][2] = b;  L[3][3] = a;
}
__device__ __forceinline__ void quat_right(const float q[4], float R[4][4]) {
  const float p = q[0], qq = q[1], r = q[2], s = q[3];
  R[0][0] = p;  R[0][1] = -qq; R[0][2] = -r;  R[0][3] = -s;
  R[1][0] = qq; R[1][1] = p;   R[1][2] = s;   R[1][3] = -r;
  R[2][0] = r;  R[2][1] = -s;  R[2][2] = p;   R[2][3] = qq;
  R[3][0] = s;  R[3][1] = r;   R[3][2] = -qq; R[3][3] = p;
}

// A1 + the temporal half of A2: activations, the TIME row of R = L(q_l) R(q_r) (eq. 8), Sigma_44, the marginal weight
// (eq. 10) and the p(t) < marginal_min filter (L324).  Returns G_VISIBLE if the primitive is alive at t; fills g.s, g.ql,
// g.qr, g.inv_nl/nr, row 3 of g.R4 / g.M, g.b, g.dt, g.w and the fp64 factors (Ld, Rd) that geom_space continues from.
// The forward preprocess calls it alone first (one thread per primitive, three primitives out of four stop here at cfg3).
struct GeomQ { double Ld[4][4], Rd[4][4]; };

#define FDGS_R_ROW(i)                                                                                                         \
  _Pragma("unroll") for (int k = 0; k < 4; ++k) {                                                                             \
    const double acc = fma(q.Ld[i][0], q.Rd[0][k], fma(q.Ld[i][1], q.Rd[1][k], fma(q.Ld[i][2], q.Rd[2][k], q.Ld[i][3] * q.Rd[3][k])));      \
    g.R4[i][k] = (float)acc; g.M[i][k] = (float)acc * g.s[k];                                                                 \
  }

__device__ __forceinline__ int geom_time(const float4 mean, const float4 ls, const float4 ql_raw, const float4 qr_raw,
                                         const float logit, const ViewParams& vp, const CfgParams& cp, Geom& g, GeomQ& q) {
  const float qlr[4] = {ql_raw.x, ql_raw.y, ql_raw.z, ql_raw.w}, qrr[4] = {qr_raw.x, qr_raw.y, qr_raw.z, qr_raw.w};
  const float lsv[4] = {ls.x, ls.y, ls.z, ls.w};
  float nl2 = 0.f, nr2 = 0.f;
#pragma unroll
  for (int k = 0; k < 4; ++k) { nl2 = fmaf(qlr[k], qlr[k], nl2); nr2 = fmaf(qrr[k], qrr[k], nr2); }
  const float chk = mean.x + mean.y + mean.z + mean.w + ls.x + ls.y + ls.z + ls.w + logit + nl2 + nr2;
  if (!isfinite(chk) || !(nl2 > 0.f) || !(nr2 > 0.f)) return G_CULL_NONFINITE;
  g.inv_nl = 1.0f / sqrtf(nl2); g.inv_nr = 1.0f / sqrtf(nr2);
#pragma unroll
  for (int k = 0; k < 4; ++k) { g.s[k] = expf(lsv[k]); g.ql[k] = qlr[k] * g.inv_nl; g.qr[k] = qrr[k] * g.inv_nr; }
  // eq. 8: R = L(q_l) R(q_r); eq. 7: Sigma = M M^T with M = R diag(s).
  // The 16 four-term dot products are taken in fp64 (~100 DFMA per primitive, nothing next to the HBM time):
  // an entry of R that is small against its terms would otherwise carry ~1e-7 ABSOLUTE error, and the time
  // row of R is multiplied by a scale s_t that is typically 30x the spatial ones, so Sigma_44 and the marginal
  // weight would lose up to two digits for nearly time-orthogonal primitives.
  // The time row of R (row 3) comes first: it alone gives Sigma_44 and hence the marginal cull, which removes three
  // primitives out of four at cfg3 before the other twelve entries are formed.  One fp64 rsqrt: the product of the
  // two normalisations scales the right factor.
  double qld[4], qrd[4];
  {
    double dl2 = 0.0, dr2 = 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) { dl2 = fma((double)qlr[k], (double)qlr[k], dl2); dr2 = fma((double)qrr[k], (double)qrr[k], dr2); }
    const double nrm = rsqrt(dl2 * dr2);
#pragma unroll
    for (int k = 0; k < 4; ++k) { qld[k] = qlr[k]; qrd[k] = qrr[k] * nrm; }
  }
  const double Ld[4][4] = {{qld[0], -qld[1], -qld[2], -qld[3]}, {qld[1], qld[0], -qld[3], qld[2]},
                           {qld[2], qld[3], qld[0], -qld[1]}, {qld[3], -qld[2], qld[1], qld[0]}};
  const double Rd[4][4] = {{qrd[0], -qrd[1], -qrd[2], -qrd[3]}, {qrd[1], qrd[0], qrd[3], -qrd[2]},
                           {qrd[2], -qrd[3], qrd[0], qrd[1]}, {qrd[3], qrd[2], -qrd[1], qrd[0]}};
#pragma unroll
  for (int r = 0; r < 4; ++r)
#pragma unroll
    for (int k = 0; k < 4; ++k) { q.Ld[r][k] = Ld[r][k]; q.Rd[r][k] = Rd[r][k]; }
  FDGS_R_ROW(3)
  // eq. 10: marginal weight, and the p(t) < marginal_min filter (L324)
  g.b = g.M[3][0] * g.M[3][0] + g.M[3][1] * g.M[3][1] + g.M[3][2] * g.M[3][2] + g.M[3][3] * g.M[3][3];
  g.dt = vp.t - mean.w;
  g.w = expf(-0.5f * g.dt * g.dt / g.b);
  if (!isfinite(g.w) || !(g.b > 0.f) || !isfinite(g.b)) return G_CULL_NONFINITE;
  if (g.w < cp.marginal_min) return G_CULL_TIME;
  return G_VISIBLE;
}

// The rest of A2 and A3 for a primitive that geom_time found alive: the other three rows of R, the slice in factor form,
// camera transform, near cull, pinhole projection, Jacobian, Sigma_2d.  Returns the status.
__device__ __forceinline__ int geom_space(const float4 mean, const float logit, const ViewParams& vp, const CfgParams& cp, Geom& g,
                                          const GeomQ& q) {
  FDGS_R_ROW(0) FDGS_R_ROW(1) FDGS_R_ROW(2)
  // eq. 9 in factor form
  const float inv_b = 1.0f / g.b;
  const float mu3[3] = {mean.x, mean.y, mean.z};
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    g.c[r] = g.M[r][0] * g.M[3][0] + g.M[r][1] * g.M[3][1] + g.M[r][2] * g.M[3][2] + g.M[r][3] * g.M[3][3];
    g.muc[r] = fmaf(g.c[r] * inv_b, g.dt, mu3[r]);
#pragma unroll
    for (int k = 0; k < 4; ++k) g.Nm[r][k] = fmaf(-g.c[r] * inv_b, g.M[3][k], g.M[r][k]);
  }
  // camera space, near cull, pinhole projection (eq. 3)
#pragma unroll
  for (int r = 0; r < 3; ++r)
    g.p[r] = fmaf(vp.W[r][0], g.muc[0], fmaf(vp.W[r][1], g.muc[1], fmaf(vp.W[r][2], g.muc[2], vp.tau[r])));
  const float z = g.p[2];
  if (!isfinite(z) || !isfinite(g.p[0]) || !isfinite(g.p[1])) return G_CULL_NONFINITE;
  if (z <= cp.znear) return G_CULL_NEAR;
  const float iz = 1.0f / z;
  const float xz = g.p[0] * iz, yz = g.p[1] * iz;
  g.u = fmaf(vp.fx, xz, vp.cx);
  g.v = fmaf(vp.fy, yz, vp.cy);
  // Jacobian at the guard-band clamped point, T = J W, B = T N
  g.clampx = fabsf(xz) > vp.limx; g.clampy = fabsf(yz) > vp.limy;
  g.xr = g.clampx ? copysignf(vp.limx, xz) : xz;
  g.yr = g.clampy ? copysignf(vp.limy, yz) : yz;
  const float j00 = vp.fx * iz, j02 = -vp.fx * g.xr * iz, j11 = vp.fy * iz, j12 = -vp.fy * g.yr * iz;
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    g.T[0][q] = fmaf(j00, vp.W[0][q], j02 * vp.W[2][q]);
    g.T[1][q] = fmaf(j11, vp.W[1][q], j12 * vp.W[2][q]);
  }
#pragma unroll
  for (int r = 0; r < 2; ++r)
#pragma unroll
    for (int k = 0; k < 4; ++k)
      g.Bm[r][k] = fmaf(g.T[r][0], g.Nm[0][k], fmaf(g.T[r][1], g.Nm[1][k], g.T[r][2] * g.Nm[2][k]));
  float n0 = 0.f, n1 = 0.f, d01 = 0.f, minors = 0.f;
#pragma unroll
  for (int k = 0; k < 4; ++k) { n0 = fmaf(g.Bm[0][k], g.Bm[0][k], n0); n1 = fmaf(g.Bm[1][k], g.Bm[1][k], n1); d01 = fmaf(g.Bm[0][k], g.Bm[1][k], d01); }
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = i + 1; j < 4; ++j) {
      const float m = g.Bm[0][i] * g.Bm[1][j] - g.Bm[0][j] * g.Bm[1][i];
      minors = fmaf(m, m, minors);
    }
  g.a2 = n0 + cp.dilation; g.c2 = n1 + cp.dilation; g.b2 = d01;
  g.det = fmaf(cp.dilation, cp.dilation + n0 + n1, minors);
  if (!(g.det > 0.f) || !isfinite(g.det)) return G_CULL_NONFINITE;
  g.sig = 1.0f / (1.0f + expf(-logit));
  g.sig_neg = 1.0f / (1.0f + expf(logit));
  return G_VISIBLE;
}
#undef FDGS_R_ROW

// Runs A1-A3 up to Sigma_2d.  Returns the status; fields are valid up to the point of the cull.
__device__ __forceinline__ int geom_forward(const float4 mean, const float4 ls, const float4 ql_raw, const float4 qr_raw,
                                            const float logit, const ViewParams& vp, const CfgParams& cp, Geom& g,
                                            const void* prefetch = nullptr, const int prefetch_bytes = 0) {
  GeomQ q;
  const int st = geom_time(mean, ls, ql_raw, qr_raw, logit, vp, cp, g, q);
  if (st != G_VISIBLE) return st;
  // the primitive is alive at t: start fetching what only survivors read (its colour block) under the arithmetic below
  if (prefetch) prefetch_l2(prefetch, prefetch_bytes);
  return geom_space(mean, logit, vp, cp, g, q);
}

// ---- real SH (degree <= 3), orthonormal, Condon-Shortley phase kept (S5) ----
#define SH_C0 0.28209479177387814f
#define SH_C1 0.4886025119029199f
#define SH_C2 1.0925484305920792f
#define SH_C20 0.31539156525252005f
#define SH_C22 0.5462742152960396f
#define SH_C3 0.5900435899266435f
#define SH_C4 2.890611442640554f
#define SH_C42 1.445305721320277f
#define SH_C5 0.4570457994644658f
#define SH_C6 0.3731763325901154f

template <int KD>
__device__ __forceinline__ void sh_basis(const float x, const float y, const float z, float* Y) {
  Y[0] = SH_C0;
  if (KD > 1) { Y[1] = -SH_C1 * y; Y[2] = SH_C1 * z; Y[3] = -SH_C1 * x; }
  if (KD > 4) {
    const float xx = x * x, yy = y * y, zz = z * z;
    Y[4] = SH_C2 * x * y; Y[5] = -SH_C2 * y * z; Y[6] = SH_C20 * (2.f * zz - xx - yy);
    Y[7] = -SH_C2 * x * z; Y[8] = SH_C22 * (xx - yy);
    if (KD > 9) {
      Y[9] = -SH_C3 * y * (3.f * xx - yy); Y[10] = SH_C4 * x * y * z; Y[11] = -SH_C5 * y * (4.f * zz - xx - yy);
      Y[12] = SH_C6 * z * (2.f * zz - 3.f * xx - 3.f * yy); Y[13] = -SH_C5 * x * (4.f * zz - xx - yy);
      Y[14] = SH_C42 * z * (xx - yy); Y[15] = -SH_C3 * x * (xx - 3.f * yy);
    }
  }
}

}  // namespace fdgs
