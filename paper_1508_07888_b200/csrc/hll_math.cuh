// hll_math.cuh -- per-cell and per-face arithmetic of the HLL interface flux (reading A19), shared by
// transport_hll.cu (dense block) and amr.cu (refined levels of the standard AMR scheme).  See transport_hll.cu for the
// derivation of the wave speeds in the internal variables phi = F / c.
#pragma once
#include "transport_math.cuh"

namespace emma {

struct Aux {                                   // closure and wave speeds of one cell
  float a, b;                                  // Pi = a I + b phi (x) phi
  float lm[3], lp[3];                          // lmin, lmax per direction, in units of c
};

__device__ __forceinline__ Aux make_aux(const float4& U)
{
  Aux A;
  const float rN = sel_ge(U.x, 1.1754944e-38f, frcp(U.x));           // A2: N <= 0 (or denormal) -> f = 0
  float rx = U.y * rN, ry = U.z * rN, rz = U.w * rN;
  const float f2raw = fmaf(rx, rx, fmaf(ry, ry, rz * rz));
  const float f2 = fminf(f2raw, 1.f);
  const float xi = fsqrt(fmaf(-3.f, f2, 4.f));
  const float i2 = frcp(2.f + xi);
  const float q = f2 * i2;
  A.a = fmaf(-U.x, q, 0.33333334f * U.x);
  A.b = sel_ge(f2raw, 1.0000001e-30f, 3.f * i2 * rN * rcp_if_gt1(f2raw));       // = 3 q / (N f^2), see closure_ab
  if (f2raw > 1.f) { const float s = rsqrtf(f2raw); rx *= s; ry *= s; rz *= s; }   // f clipped to 1: r -> unit vector
  const float k = 2.f * (1.f - f2) * frcp(xi + 1.f), ixi = frcp(xi), t3 = 3.f * i2;
  const float sx = fsqrt(fmaxf(k * fmaf(-t3 * rx, rx, xi), 0.f));
  const float sy = fsqrt(fmaxf(k * fmaf(-t3 * ry, ry, xi), 0.f));
  const float sz = fsqrt(fmaxf(k * fmaf(-t3 * rz, rz, xi), 0.f));
  A.lm[0] = (rx - sx) * ixi; A.lp[0] = (rx + sx) * ixi;
  A.lm[1] = (ry - sy) * ixi; A.lp[1] = (ry + sy) * ixi;
  A.lm[2] = (rz - sz) * ixi; A.lp[2] = (rz + sz) * ixi;
  return A;
}

// packed helpers (sm_100a FADD2 / FMUL2 / FFMA2 on register pairs)
__device__ __forceinline__ void sub2(float& dx, float& dy, float ax, float ay, float bx, float by)
{
  fma2(dx, dy, bx, by, -1.f, -1.f, ax, ay);
}

// flux vector G_d of a cell and the HLL combination for the face between L (towards -d) and R (towards +d):
// H = wl G_L + wr G_R + wd (U_R - U_L), evaluated on the (N, phi_x) and (phi_y, phi_z) halves with packed arithmetic
template <int D>
__device__ __forceinline__ float4 hll_face(const float4& UL, float aL, float bL, float lmL, float lpL,
                                           const float4& UR, float aR, float bR, float lmR, float lpR)
{
  const float pL = comp<D>(UL), pR = comp<D>(UR);
  const float uL = bL * pL, uR = bR * pR;
  float4 GL, GR;
  GL.x = pL; GL.y = uL * UL.y; mul2(GL.z, GL.w, UL.z, UL.w, uL, uL);
  GR.x = pR; GR.y = uR * UR.y; mul2(GR.z, GR.w, UR.z, UR.w, uR, uR);
  if (D == 0) { GL.y += aL; GR.y += aR; } else if (D == 1) { GL.z += aL; GR.z += aR; } else { GL.w += aL; GR.w += aR; }
  const float lp = fmaxf(0.f, fmaxf(lpL, lpR)), lm = fminf(0.f, fminf(lmL, lmR));
  const float den = lp - lm;
  // l+ = l- = 0 (both cells stream exactly along the face): G vanishes there too and H = 0.  The guard also covers a
  // denormal den (transverse speeds of ~1e-38 from rounding dust in phi), whose approximate reciprocal is inf
  const float inv = (den > 1e-20f) ? frcp(den) : 0.f;
  const float wl = lp * inv, wr = -lm * inv, wd = lp * lm * inv;
  float4 H, dU;
  sub2(dU.x, dU.y, UR.x, UR.y, UL.x, UL.y); sub2(dU.z, dU.w, UR.z, UR.w, UL.z, UL.w);
  mul2(H.x, H.y, dU.x, dU.y, wd, wd); mul2(H.z, H.w, dU.z, dU.w, wd, wd);
  fma2(H.x, H.y, GR.x, GR.y, wr, wr, H.x, H.y); fma2(H.z, H.w, GR.z, GR.w, wr, wr, H.z, H.w);
  fma2(H.x, H.y, GL.x, GL.y, wl, wl, H.x, H.y); fma2(H.z, H.w, GL.z, GL.w, wl, wl, H.z, H.w);
  return H;
}

// closure and the wave speeds of ONE direction (a face needs nothing else of its neighbour)
struct AuxD { float a, b, lm, lp; };

__device__ __forceinline__ AuxD make_aux_dir(const float4& U, int d)
{
  AuxD A;
  const float rN = sel_ge(U.x, 1.1754944e-38f, frcp(U.x));
  float rx = U.y * rN, ry = U.z * rN, rz = U.w * rN;
  const float f2raw = fmaf(rx, rx, fmaf(ry, ry, rz * rz));
  const float f2 = fminf(f2raw, 1.f);
  const float xi = fsqrt(fmaf(-3.f, f2, 4.f));
  const float i2 = frcp(2.f + xi);
  const float q = f2 * i2;
  A.a = fmaf(-U.x, q, 0.33333334f * U.x);
  A.b = sel_ge(f2raw, 1.0000001e-30f, 3.f * i2 * rN * rcp_if_gt1(f2raw));
  float rd = (d == 0) ? rx : (d == 1) ? ry : rz;
  if (f2raw > 1.f) rd *= rsqrtf(f2raw);
  const float k = 2.f * (1.f - f2) * frcp(xi + 1.f), ixi = frcp(xi), t3 = 3.f * i2;
  const float sd = fsqrt(fmaxf(k * fmaf(-t3 * rd, rd, xi), 0.f));
  A.lm = (rd - sd) * ixi; A.lp = (rd + sd) * ixi;
  return A;
}
__device__ __forceinline__ AuxD aux_dir(const Aux& X, int d)
{
  AuxD A;
  A.a = X.a; A.b = X.b; A.lm = X.lm[d]; A.lp = X.lp[d];
  return A;
}

}  // namespace emma
