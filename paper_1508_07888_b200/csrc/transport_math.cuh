// transport_math.cuh -- per-cell arithmetic of the M1 transport update shared by the transport kernels
// (closure Eq. 22-23 with readings A1/A2, the U -/+ G_d neighbour contributions of Eq. 30 + 32, boundary index map A13).
// See transport.cu for the derivation of the update in the internal variables phi = F / c.
#pragma once
#include "emma_rt_internal.cuh"

namespace emma {

// packed fp32 (sm_100a FFMA2 / FADD2): d = a * b + c on a register pair
__device__ __forceinline__ void fma2(float& dx, float& dy, float ax, float ay, float bx, float by, float cx, float cy)
{
  asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\t"
      "mov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
      "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(dx), "=f"(dy)
      : "f"(ax), "f"(ay), "f"(bx), "f"(by), "f"(cx), "f"(cy));
}
__device__ __forceinline__ void mul2(float& dx, float& dy, float ax, float ay, float bx, float by)
{
  asm("{\n\t.reg .b64 ra, rb, rd;\n\t"
      "mov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
      "mul.rn.f32x2 rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(dx), "=f"(dy)
      : "f"(ax), "f"(ay), "f"(bx), "f"(by));
}

// L2 prefetch of one cell (no register or shared-memory cost): the march's own load of that cell, a few planes
// later, then hits L2 instead of waiting a full DRAM round trip
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }

// d = (x >= lo) ? v : 0 as a predicated select: keeps the closure branch-free (the compiler otherwise branches
// around the MUFU ops, which chops the march into basic blocks and serialises the shared-memory latencies)
__device__ __forceinline__ float sel_ge(float x, float lo, float v)
{
  float d;
  asm("{\n\t.reg .pred p;\n\tsetp.ge.f32 p, %1, %2;\n\tselp.f32 %0, %3, 0f00000000, p;\n\t}" : "=f"(d) : "f"(x), "f"(lo), "f"(v));
  return d;
}

// 1 / x when x > 1, else 1 (the reciprocal is issued under the predicate)
__device__ __forceinline__ float rcp_if_gt1(float x)
{
  float d;
  asm("{\n\t.reg .pred p;\n\tsetp.gt.f32 p, %1, 0f3F800000;\n\tmov.f32 %0, 0f3F800000;\n\t@p rcp.approx.ftz.f32 %0, %1;\n\t}" : "=f"(d) : "f"(x));
  return d;
}

__device__ __forceinline__ void closure_ab(const float4& U, float& a, float& b)
{
  // A2: N <= 0 -> f = 0.  A denormal N (light that has just reached a dark cell) counts as 0: rcp.ftz of it is inf.
  const float rN = sel_ge(U.x, 1.1754944e-38f, frcp(U.x));
  const float rx = U.y * rN, ry = U.z * rN, rz = U.w * rN;
  const float f2raw = fmaf(rx, rx, fmaf(ry, ry, rz * rz));
  const float f2 = fminf(f2raw, 1.f);          // A2: f clipped to [0,1]
  const float s = fsqrt(fmaf(-3.f, f2, 4.f));
  const float r2s = frcp(2.f + s);
  const float q = f2 * r2s;
  a = fmaf(-U.x, q, 0.33333334f * U.x);
  // b = 3 q / (N f^2) = 3 / ((2 + s) N) * (f2 / f2raw): the last factor is 1 unless f was clipped (rare), so the
  // reciprocal of f2raw is predicated on the clip and costs no MUFU cycle otherwise.
  // A1: |F| = 0 -> no n(x)n term; below f^2 = 1e-30 the term (<= f^2 N) is far under fp32 resolution of a
  // (f2raw is +inf or NaN only for non-finite inputs, which the diagnostics report)
  b = sel_ge(f2raw, 1.0000001e-30f, 3.f * r2s * rN * rcp_if_gt1(f2raw));
}

// map an index that may be one cell outside [0,n) through the boundary condition of that face (A13)
__device__ __forceinline__ int bc_map(int i, int n, int bc_lo, int bc_hi, bool& flip)
{
  flip = false;
  if (i < 0) {
    if (bc_lo == EMMA_RT_BC_PERIODIC) return i + n;
    flip = (bc_lo == EMMA_RT_BC_REFLECTIVE);
    return 0;
  }
  if (i >= n) {
    if (bc_hi == EMMA_RT_BC_PERIODIC) return i - n;
    flip = (bc_hi == EMMA_RT_BC_REFLECTIVE);
    return n - 1;
  }
  return i;
}

template <int D>
__device__ __forceinline__ float comp(const float4& U) { return (D == 0) ? U.y : (D == 1) ? U.z : U.w; }

// contribution of the neighbour on the + side of direction d:  U - G_d = (N - phi_d, phi (1 - b phi_d) - a e_d)
template <int D>
__device__ __forceinline__ void add_plus(float4& acc, const float4& U, float a, float b)
{
  const float pd = comp<D>(U);
  const float u = fmaf(-b, pd, 1.f);
  fma2(acc.x, acc.y, U.x, U.y, 1.f, u, acc.x, acc.y);
  fma2(acc.z, acc.w, U.z, U.w, u, u, acc.z, acc.w);
  acc.x -= pd;
  if (D == 0) acc.y -= a; else if (D == 1) acc.z -= a; else acc.w -= a;
}
// neighbour on the - side:  U + G_d
template <int D>
__device__ __forceinline__ void add_minus(float4& acc, const float4& U, float a, float b)
{
  const float pd = comp<D>(U);
  const float u = fmaf(b, pd, 1.f);
  fma2(acc.x, acc.y, U.x, U.y, 1.f, u, acc.x, acc.y);
  fma2(acc.z, acc.w, U.z, U.w, u, u, acc.z, acc.w);
  acc.x += pd;
  if (D == 0) acc.y += a; else if (D == 1) acc.z += a; else acc.w += a;
}
// the same, starting a fresh accumulator (no add of the old value)
__device__ __forceinline__ float4 below_z(const float4& U, float a, float b)
{
  const float u = fmaf(b, U.w, 1.f);
  float4 r;
  r.x = U.x + U.w;
  r.y = U.y * u;
  mul2(r.z, r.w, U.z, U.w, u, u);
  r.w += a;
  return r;
}

}  // namespace emma
