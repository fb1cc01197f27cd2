// chem_math.cuh -- per-cell arithmetic of the sub-cycled thermo-chemistry (Eq. 43-48, readings A5-A12), shared by the
// chemistry kernels (chemistry.cu) and the fused transport -> chemistry pass (fused.cu).  See chemistry.cu for the
// conditioning notes (x and 1-x both carried, per-atom energies, rates through lg2/ex2).
#pragma once
#include "emma_rt_internal.cuh"
#include "transport_math.cuh"

namespace emma {

constexpr float KB15 = 1.5f * 1.380649e-16f;          // (3/2) k_B  [erg/K]   (A10: e = (3/2)(1+x) n0 k_B T)
constexpr float LOG2E = 1.4426950408889634f;
constexpr float FINF = __builtin_huge_valf();

template <int G>
struct CellState {
  float N[G], px[G], py[G], pz[G];
  float S[G];
  float n0, x, y, eps;
};

struct Rates { float alpha, beta, cHI, cHII, rec; };

// per-cell tallies, folded into the thread's fp64 Acc when the cell completes
struct CellTally { float absorbed = 0.f, injected = 0.f, recomb = 0.f; unsigned nsub = 0, nhalv = 0; };

__device__ __forceinline__ void decode_x(float xs, float& x, float& y)
{
  if (__float_as_int(xs) < 0) { y = -xs; x = 1.f - y; } else { x = xs; y = 1.f - xs; }
}
__device__ __forceinline__ float encode_x(float x, float y)
{
  return (x <= 0.5f) ? fabsf(x) : __int_as_float(__float_as_int(fabsf(y)) | 0x80000000);
}

// A11 rate fits at temperature T.  lam = 2 * 157807 / T.
__device__ __forceinline__ Rates rates_at(float T, int otsa, float x, float n0)
{
  Rates r;
  const float lT = flg2(T), rT = frcp(T);
  const float llam = 18.267802f - lT;                 // log2(315614 / T)
  const float lam = 315614.f * rT;
  // alpha_B = 2.753e-14 lam^1.5 / (1 + (lam/2.740)^0.407)^2.242
  const float aB = 2.753e-14f * fex2(1.5f * llam - 2.242f * flg2(1.f + fex2(0.407f * (llam - 1.4541759f))));
  // beta = 21.11 T^-1.5 e^{-lam/2} lam^-1.089 / (1 + (lam/0.354)^0.874)^1.101
  const float be = 21.11f * fex2(-1.5f * lT - 1.089f * llam - 1.101f * flg2(1.f + fex2(0.874f * (llam + 1.4981787f)))) *
                   fex2(-0.5f * LOG2E * lam);
  const float sqT = fsqrt(T);
  // collisional excitation + collisional ionisation cooling, per n_e n_HI
  r.cHI = 7.5e-19f * fex2(-118348.f * LOG2E * rT) * frcp(1.f + sqT * 3.1622776e-3f) + 2.179e-11f * be;
  const float dl = 5.5f - 0.30103f * lT;              // 5.5 - log10 T
  const float ff = 1.42e-27f * (1.1f + 0.34f * fex2(-(LOG2E / 3.f) * dl * dl)) * sqT;     // bremsstrahlung
  r.beta = be;
  if (otsa) {
    // Lambda_rec,B = 3.435e-30 T lam^1.970 / (1 + (lam/2.250)^0.376)^3.720
    const float recB = 3.435e-30f * T * fex2(1.970f * llam - 3.720f * flg2(1.f + fex2(0.376f * (llam - 1.169925f))));
    r.alpha = aB;                                     // alpha_A := alpha_B
    r.cHII = recB + ff;
    r.rec = 0.f;
  } else {
    const float aA = 1.269e-13f * fex2(1.503f * llam - 1.923f * flg2(1.f + fex2(0.470f * (llam + 0.9378783f))));
    const float recA = 1.778e-29f * T * fex2(1.965f * llam - 2.697f * flg2(1.f + fex2(0.502f * (llam + 0.8862995f))));
    r.alpha = aA;
    r.cHII = recA + ff;
    r.rec = (aA - aB) * x * x * n0 * n0;              // A6: recombination radiation, group 1 only
  }
  return r;
}

// First guess of the chemical step, abs(e / (H - Lambda)) (reading A9), `if_zero` when H = Lambda.  d is
// (H - Lambda) per atom at state p.  One approximate reciprocal instead of an IEEE division: the guess only picks the
// starting dtau of the halving loop and feeds the dtau_min diagnostic (held to 1e-3 against the oracle).
__device__ __forceinline__ float first_guess(float eps, float d, float if_zero)
{
  const float ad = fabsf(d);
  return (ad == 0.f) ? if_zero : fabsf(eps) * frcp(ad);
}

// Eq. 44 with the factor chosen by attempt(): m > 0 -> F' = F m (m = 1/(1 + k dtau), strong sink);
// m <= 0 -> F' = F + F m (m = -k dtau/(1 + k dtau), weak sink: only the small decrement is rounded)
__device__ __forceinline__ float decay(float v, float m) { return (m > 0.f) ? v * m : fmaf(v, m, v); }

// One attempt of Eq. 43-48 with step dtau from state p = c.  Returns the 10 % verdict.
template <int G>
__device__ __forceinline__ bool attempt(const ChemParams& cp, const CellState<G>& c, const Rates& r, float dtau,
                                        float (&N1)[G], float (&iden)[G], float& x1, float& y1, float& eps1)
{
  // Every backward-Euler quotient q' = (q + a dtau)/(1 + k dtau) is evaluated in the form that loses nothing:
  // for a weak sink (k dtau <= 1/2) as the increment q + (a dtau - k dtau q)/(1 + k dtau), whose rounding is
  // relative to the (small) increment, so a slowly relaxing cell does not drift by an ulp per step; for a strong
  // sink as the printed quotient (the increment form would cancel there).
  const float k = c.y * c.n0 * dtau;
  float ion = 0.f, hsum = 0.f;
#pragma unroll
  for (int g = 0; g < G; g++) {
    const float kd = cp.csig[g] * k;                                  // A5: c sigma (1-x^p) n0 dtau
    const float id = frcp(1.f + kd);
    const float kid = kd * id;
    const float sdt = (c.S[g] + (g == 0 ? r.rec : 0.f)) * dtau;
    const bool strong = kd > 0.5f;
    N1[g] = strong ? (c.N[g] + sdt) * id : c.N[g] + fmaf(-kid, c.N[g], sdt * id);     // Eq. 43
    iden[g] = strong ? id : -kid;                                     // Eq. 44, applied on commit by decay()
    ion = fmaf(cp.csig[g], N1[g], ion);                               // Eq. 41
    hsum = fmaf(cp.csigE[g], N1[g], hsum);                            // Eq. 42
  }
  const float Gt = dtau * fmaf(r.beta * c.x, c.n0, ion);
  const float rr = r.alpha * c.x * c.x * c.n0 * dtau;
  const float inv = frcp(1.f + Gt);
  float xa, ya;
  if (Gt > 0.5f) {
    xa = (c.x + (Gt - rr)) * inv;                                     // Eq. 45, solved for x
    ya = (c.y + rr) * inv;                                            // Eq. 45 as printed (1 - x^{p+1})
  } else {
    const float dx = fmaf(Gt, c.y, -rr) * inv;                        // x' - x
    xa = c.x + dx;
    ya = c.y - dx;
  }
  if (xa <= 0.5f) ya = 1.f - xa; else xa = 1.f - ya;
  xa = fminf(fmaxf(xa, 0.f), 1.f);                                    // guards (A7)
  ya = fminf(fmaxf(ya, 0.f), 1.f);
  x1 = xa; y1 = ya;
  if (!cp.thermal) {                                                  // isothermal test mode: T held (A9)
    const float dx = (xa <= 0.5f) ? xa - c.x : c.y - ya;
    eps1 = fmaf(c.eps * dx, frcp(1.f + c.x), c.eps);
    return true;
  }
  // Eq. 46-48 per atom: heating c (1-x') sum Sigma_E N', cooling Lambda(n0, x', T^p)/n0
  const float de = dtau * (ya * hsum - c.n0 * xa * fmaf(ya, r.cHI, xa * r.cHII));
  eps1 = c.eps + de;
  return (fabsf(de) <= cp.e_tol * c.eps) && (eps1 > 0.f);
}

// One ACCEPTED sub-step (rates at state p, first guess, halvings).  Returns false on ESUBCYCLE.
template <int G>
__device__ __forceinline__ bool substep(const ChemParams& cp, CellState<G>& c, float& rem, CellTally& tl, float& dtau_min)
{
  const float T = c.eps * frcp(KB15 * (1.f + c.x));
  const Rates r = rates_at(T, cp.otsa, c.x, c.n0);
  float dtau = rem;
  if (cp.thermal) {
    float hsum = 0.f;
#pragma unroll
    for (int g = 0; g < G; g++) hsum = fmaf(cp.csigE[g], c.N[g], hsum);
    const float d = c.y * hsum - c.n0 * c.x * fmaf(c.y, r.cHI, c.x * r.cHII);      // (H - Lambda)/n0 at state p
    const float guess = first_guess(c.eps, d, rem);                                 // PAPER.md:290 (A9: abs)
    dtau_min = fminf(dtau_min, guess);
    dtau = fminf(rem, guess);
  }
  float N1[G], iden[G], x1, y1, eps1;
  unsigned halv = 0;
  bool ok = true;
  while (!attempt<G>(cp, c, r, dtau, N1, iden, x1, y1, eps1)) {
    if (halv >= (unsigned)cp.max_halvings) { ok = false; break; }
    dtau *= 0.5f;                                                     // PAPER.md:312 "divided by 2"
    halv++;
  }
  tl.nhalv += halv;
  if (!ok) return false;
  const float k = c.y * c.n0 * dtau;
#pragma unroll
  for (int g = 0; g < G; g++) {
    tl.absorbed = fmaf(cp.csig[g] * k, N1[g], tl.absorbed);           // A15: the sink of Eq. 43
    tl.injected = fmaf(c.S[g], dtau, tl.injected);
    c.N[g] = N1[g];
    c.px[g] = decay(c.px[g], iden[g]); c.py[g] = decay(c.py[g], iden[g]); c.pz[g] = decay(c.pz[g], iden[g]);   // Eq. 44
  }
  tl.recomb = fmaf(r.rec, dtau, tl.recomb);
  c.x = x1; c.y = y1; c.eps = eps1;
  tl.nsub++;
  rem = (dtau >= rem) ? 0.f : rem - dtau;
  if (tl.nsub >= EMMA_RT_MAX_SUBSTEPS && rem > 0.f) return false;
  return true;
}

// dV_total: the volume used for the photon total (= dV, or 0 when this sweep is not the one that counts the photons of its
// level: a refined level of the standard AMR scheme is swept 2^l times per coarse step)
__device__ __forceinline__ void fold(Acc& a, const CellTally& tl, const float* N, int G, double dV, double dV_total)
{
  a.absorbed += (double)tl.absorbed * dV;
  a.injected += (double)tl.injected * dV;
  a.recomb += (double)tl.recomb * dV;
  a.nsub += tl.nsub; a.nhalv += tl.nhalv;
  a.nsub_max = max(a.nsub_max, tl.nsub);
  float s = 0.f;
  for (int g = 0; g < G; g++) s += N[g];
  a.total += (double)s * dV_total;
}

template <int G>
__device__ __forceinline__ void load_sources(const LevelDev& L, long long cell, float (&S)[G])
{
#pragma unroll
  for (int g = 0; g < G; g++) S[g] = 0.f;
  if (L.n_src == 0) return;
  if (!((L.srcmask[cell >> 5] >> (cell & 31)) & 1u)) return;
  int lo = 0, hi = L.n_src - 1;                                       // sorted list, the cell is in it
  const int key = (int)cell;
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (L.src_cell[mid] < key) lo = mid + 1; else hi = mid;
  }
#pragma unroll
  for (int g = 0; g < G; g++) S[g] = L.src_S[(size_t)lo * G + g];
}

// the same with the cell's word of the source bitmap already loaded
template <int G>
__device__ __forceinline__ void load_sources_word(const LevelDev& L, long long cell, unsigned word, float (&S)[G])
{
#pragma unroll
  for (int g = 0; g < G; g++) S[g] = 0.f;
  if (!((word >> (cell & 31)) & 1u)) return;
  int lo = 0, hi = L.n_src - 1;
  const int key = (int)cell;
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (L.src_cell[mid] < key) lo = mid + 1; else hi = mid;
  }
#pragma unroll
  for (int g = 0; g < G; g++) S[g] = L.src_S[(size_t)lo * G + g];
}

template <int G>
__device__ __forceinline__ void load_cell(const LevelDev& L, long long cell, const float4* __restrict__ U,
                                          long long ustride, long long ucell, CellState<G>& c)
{
#pragma unroll
  for (int g = 0; g < G; g++) {
    const float4 u = U[(size_t)g * ustride + ucell];
    c.N[g] = u.x; c.px[g] = u.y; c.py[g] = u.z; c.pz[g] = u.w;
  }
  c.n0 = L.n0[cell];
  c.eps = L.eps[cell];
  decode_x(L.xs[cell], c.x, c.y);
  load_sources<G>(L, cell, c.S);
}

// 0 * v is +-0 for a finite v and NaN for an infinite or NaN v, so one packed FMA per pair of values accumulates
// "anything non-finite" into s (IEEE arithmetic: nothing here is folded away without fast-math)
template <int G>
__device__ __forceinline__ bool finite_cell(const CellState<G>& c)
{
  float s0 = 0.f, s1 = 0.f;
  fma2(s0, s1, c.eps, c.x, 0.f, 0.f, s0, s1);
#pragma unroll
  for (int g = 0; g < G; g++) {
    fma2(s0, s1, c.N[g], c.px[g], 0.f, 0.f, s0, s1);
    fma2(s0, s1, c.py[g], c.pz[g], 0.f, 0.f, s0, s1);
  }
  return (s0 + s1) == 0.f;
}

template <int G>
__device__ __forceinline__ void store_cell(const LevelDev& L, long long cell, float4* __restrict__ U, long long ustride,
                                           const CellState<G>& c, const CellTally& tl, int record)
{
#pragma unroll
  for (int g = 0; g < G; g++) U[(size_t)g * ustride + cell] = make_float4(c.N[g], c.px[g], c.py[g], c.pz[g]);
  L.xs[cell] = encode_x(c.x, c.y);
  L.eps[cell] = c.eps;
  if (record) L.subc[cell] = min(tl.nsub, 65535u) | (min(tl.nhalv, 65535u) << 16);
}

}  // namespace emma
