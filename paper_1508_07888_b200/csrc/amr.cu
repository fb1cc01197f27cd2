// amr.cu -- standard (non-CRTA) AMR transport on refined levels (reading A21;
// PAPER.md:327-355 Eq. 49-51 / Fig. 2-3, PAPER.md:436 resolution jumps).
//
// The host (api.cu) runs the recursion advance(l, dt) = [advance(l+1, dt/2) x 2] -> transport(l) -> chemistry(l) ->
// restriction(l+1 -> l).  This file holds the kernels of one level:
//   * amr_transport_kernel: Eq. 30 + 32 for the LEAF cells of a refined level, one thread per cell and all G groups.
//     Neighbours come from the oct structure the paper describes (each oct points to the 6 cells of the
//     level below that surround its parent cell): the host keeps those pointers (`nbr`, also in the arena) and derives
//     from them, once for the static mesh, what the kernels read: the same-level neighbour oct of every oct side (`nbo`),
//     the list of faces towards a coarser leaf with their six resolved coarse references, the leaves that receive
//     deposits.  Siblings sit in the same 128-byte oct record and are exchanged by warp shuffles.  A face towards a split
//     cell computes nothing (the fine cells behind it deposit).
//   * amr_ghost_faces_kernel: the faces towards a coarser leaf, one thread per face from a host-built list, BEFORE the
//     per-cell kernel of the sweep and from start-of-step states only: MinMod-limited linear ghost, flux, and two kinds of
//     records -- the fine cell's change (one per face; the per-cell kernel adds its cell's <= 3 records to its result in
//     the order x, y, z) and what the oct side hands to the coarse leaf (one per (oct, face), the two sub-steps summed by
//     the thread that owns the side; the leaf gathers its <= 6 records in face order when its own step comes).  No
//     read-modify-write of a state buffer and no atomics: the mode is bit-reproducible.
//   * level 0 keeps the dense TMA kernel (transport_tma.cu) for the whole block; amr_fix0_kernel then recomputes the
//     (few) leaves that touch a split cell without the faces towards it and adds what the fine cells deposited: the
//     regular block stays on the bandwidth-bound kernel, the irregular part is a sparse second pass.
//   * amr_chem_kernel: Eq. 43-48 in place on the leaves of a refined level (chem_math.cuh, same arithmetic as CRTA's).
//   * restriction, initial injection, sources with chemistry off, outflow of level 0.
#include "chem_math.cuh"
#include "hll_math.cuh"
#include "transport_math.cuh"

#ifndef AMR_T_CTAS
#define AMR_T_CTAS 6
#endif

namespace emma {
namespace {

// kind: 0 a leaf of the same level, 1 a split cell of the same level, 2 a leaf of the level below (coarser),
//       3 box ghost = the cell itself (flip >= 0: that flux component inverted, A13), 4 inflow ghost (A20)
struct NbRef { int kind, lvl, flip, face; long long cell; };

__device__ __forceinline__ NbRef box_ghost(int bc, int a, int side, int lvl, long long self)
{
  NbRef r;
  r.lvl = lvl; r.cell = self; r.face = 2 * a + side; r.flip = -1;
  if (bc == EMMA_RT_BC_INFLOW) r.kind = 4;
  else { r.kind = 3; if (bc == EMMA_RT_BC_REFLECTIVE) r.flip = a; }
  return r;
}

// neighbour of a level-0 cell by coordinates
__device__ NbRef nb_ref0(const AmrDev& A, long long cell, int a, int side)
{
  const int n = A.n;
  const unsigned uc = (unsigned)cell, t = uc / (unsigned)n;          // n^3 < 2^32 (n <= 1290)
  const int i = (int)(uc % (unsigned)n), j = (int)(t % (unsigned)n), k = (int)(t / (unsigned)n);
  int ca = (a == 0) ? i : (a == 1) ? j : k;
  const long long stride = (a == 0) ? 1 : (a == 1) ? n : (long long)n * n;
  const int cn = ca + (side ? 1 : -1);
  long long nb;
  if (cn < 0 || cn >= n) {
    const int bc = A.bc[2 * a + side];
    if (bc != EMMA_RT_BC_PERIODIC) return box_ghost(bc, a, side, 0, cell);
    nb = cell + (side ? -(long long)(n - 1) : (long long)(n - 1)) * stride;
  } else nb = cell + (side ? stride : -stride);
  NbRef r;
  r.lvl = 0; r.cell = nb; r.flip = -1; r.face = 0;
  r.kind = (A.child[0] && A.child[0][nb] >= 0) ? 1 : 0;
  return r;
}

__device__ __forceinline__ float4 nb_load(const AmrDev& A, const NbRef& r, int g, const float4& self)
{
  if (r.kind == 4) return A.inflow[r.face][g];
  if (r.kind == 3) {
    float4 u = self;
    if (r.flip == 0) u.y = -u.y; else if (r.flip == 1) u.z = -u.z; else if (r.flip == 2) u.w = -u.w;
    return u;
  }
  return A.U[r.lvl][(size_t)g * A.ncell[r.lvl] + r.cell];
}

__device__ __forceinline__ float minmod(float a, float b)
{
  if (a * b <= 0.f) return 0.f;
  return (fabsf(a) < fabsf(b)) ? a : b;
}

// G_a(U) = (phi_a, a e_a + b phi_a phi): the flux vector of direction a in units of c_red (closure_ab: P = a I + b phi(x)phi)
__device__ __forceinline__ float4 flux_vec(const float4& U, float ca, float cb, int a)
{
  const float pa = (a == 0) ? U.y : (a == 1) ? U.z : U.w;
  const float t = cb * pa;
  float4 Gv = make_float4(pa, t * U.y, t * U.z, t * U.w);
  if (a == 0) Gv.y += ca; else if (a == 1) Gv.z += ca; else Gv.w += ca;
  return Gv;
}

// change of the cell (state Ui, closure ai/bi) caused by the Eq. 32 flux through its face (a, side) towards state Un:
//   + face: -nu F^ = -(nu/2) [(G_i + U_i) + (G_n - U_n)];   - face: +(nu/2) [(G_n + U_n) + (G_i - U_i)]
__device__ __forceinline__ float4 face_change_pre(int a, int side, const float4& Ui, float ai, float bi, const float4& Un,
                                                 float an, float bn, float nuh)
{
  const float4 Gi = flux_vec(Ui, ai, bi, a), Gn = flux_vec(Un, an, bn, a);
  float4 r;
  if (side) {
    r.x = -nuh * ((Gi.x + Ui.x) + (Gn.x - Un.x)); r.y = -nuh * ((Gi.y + Ui.y) + (Gn.y - Un.y));
    r.z = -nuh * ((Gi.z + Ui.z) + (Gn.z - Un.z)); r.w = -nuh * ((Gi.w + Ui.w) + (Gn.w - Un.w));
  } else {
    r.x = nuh * ((Gn.x + Un.x) + (Gi.x - Ui.x)); r.y = nuh * ((Gn.y + Un.y) + (Gi.y - Ui.y));
    r.z = nuh * ((Gn.z + Un.z) + (Gi.z - Ui.z)); r.w = nuh * ((Gn.w + Un.w) + (Gi.w - Ui.w));
  }
  return r;
}
__device__ __forceinline__ float4 face_change(int a, int side, const float4& Ui, float ai, float bi, const float4& Un, float nuh)
{
  float an, bn;
  closure_ab(Un, an, bn);
  return face_change_pre(a, side, Ui, ai, bi, Un, an, bn, nuh);
}

// position of child k among the 4 cells of its oct's side across axis a, in the order of the host-built face list
// (k increasing with bit a fixed): the bits of k without bit a
__device__ __forceinline__ int side_pos(int k, int a)
{
  return (a == 0) ? (k >> 1) : (a == 1) ? (((k >> 2) << 1) | (k & 1)) : (k & 3);
}

// What the fine cells behind face f of a leaf of level l handed to it during the two sub-steps of level l + 1 (Fig. 3 (i)-(ii)):
// `o2` is the oct of level l + 1 that fills the split neighbour; its side facing back (f ^ 1) looks at a coarser leaf -- this
// one.  The records are indexed by (oct, face) of the fine level and hold the sum of the two sub-steps (first + second, added by
// the one thread that owns the side in amr_ghost_faces_kernel).
template <int G>
__device__ __forceinline__ void gather_side(const AmrDev& A, int l, int o2, int f, float4 (&sum)[G])
{
  const size_t s = (size_t)o2 * 6 + (f ^ 1);
  const float4* __restrict__ R = A.depS[l + 1];
  const size_t cap = (size_t)A.scap[l + 1];
#pragma unroll
  for (int g = 0; g < G; g++) {
    const float4 r = R[(size_t)g * cap + s];
    sum[g].x += r.x; sum[g].y += r.y; sum[g].z += r.z; sum[g].w += r.w;
  }
}

// ---- HLL variant (reading A19) of the refined-level kernels: face by face, no cancellation algebra ------------------
// change of the cell (state Ui) caused by the HLL flux through its face (a, side) towards state Un: -/+ nu H
__device__ __forceinline__ float4 hll_change(int a, int side, const float4& Ui, const AuxD& Xi, const float4& Un, const AuxD& Xn, float nu)
{
  const float4& UL = side ? Ui : Un;
  const float4& UR = side ? Un : Ui;
  const AuxD& XL = side ? Xi : Xn;
  const AuxD& XR = side ? Xn : Xi;
  float4 H;
  if (a == 0) H = hll_face<0>(UL, XL.a, XL.b, XL.lm, XL.lp, UR, XR.a, XR.b, XR.lm, XR.lp);
  else if (a == 1) H = hll_face<1>(UL, XL.a, XL.b, XL.lm, XL.lp, UR, XR.a, XR.b, XR.lm, XR.lp);
  else H = hll_face<2>(UL, XL.a, XL.b, XL.lm, XL.lp, UR, XR.a, XR.b, XR.lm, XR.lp);
  const float w = side ? -nu : nu;
  return make_float4(w * H.x, w * H.y, w * H.z, w * H.w);
}
// A19: keep the state realizable, |phi| <= max(N, 0)
__device__ __forceinline__ void realizable(float4& U)
{
  const float f2 = fmaf(U.y, U.y, fmaf(U.z, U.z, U.w * U.w));
  const float lim = fmaxf(U.x, 0.f);
  if (f2 > lim * lim) { const float s = lim * rsqrtf(f2); U.y *= s; U.z *= s; U.w *= s; }
}

// Eq. 30 with the HLL flux on the leaves of a refined level: the layout of amr_transport_kernel (8 lanes = one oct, sibling
// states by shuffle, outer faces through nbo), every face evaluated explicitly.  The realizability limiter is applied by
// the kernel that follows (chemistry or sources), after the ghost-face kernel has added its faces.
template <int G>
__global__ void __launch_bounds__(128)
amr_transport_hll_kernel(const AmrDev A, int l, float nuh, float4* __restrict__ Unew, double dV, Partial* __restrict__ parts)
{
  Acc acc;
  const float nu = 2.f * nuh;
  const long long ncell = A.ncell[l];
  const float4* __restrict__ Ul = A.U[l];
  const int* __restrict__ child = (l < A.nl) ? A.child[l] : nullptr;
  const int* __restrict__ nbo = A.nbo[l];
  const long long span = (long long)gridDim.x * blockDim.x;
  for (long long base = (long long)blockIdx.x * blockDim.x; base < ncell; base += span) {
    const long long cell = base + threadIdx.x;
    const bool valid = cell < ncell;
    const bool leaf = valid && !(child && child[cell] >= 0);
    const bool hd = leaf && l < A.nl && ((A.hasdep[l][cell >> 5] >> (cell & 31)) & 1u);
    const int k = (int)(cell & 7);
    const long long oct = cell >> 3;
    // what the finer level deposited into this leaf (only leaves next to a split cell of their own level: host bitmap)
    float4 dsum[G];
#pragma unroll
    for (int g = 0; g < G; g++) dsum[g] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (hd) {
#pragma unroll
      for (int a = 0; a < 3; a++) {
        const int bit = (k >> a) & 1;
        const int chs = child[cell ^ (1 << a)];                       // sibling across a
        if (chs >= 0) gather_side<G>(A, l, chs, 2 * a + (1 - bit), dsum);
        const int no = nbo[oct * 6 + 2 * a + bit];
        if (no >= 0) {
          const int cho = child[(((long long)no << 3) | (k ^ (1 << a)))];
          if (cho >= 0) gather_side<G>(A, l, cho, 2 * a + bit, dsum);
        }
      }
    }
#pragma unroll
    for (int g = 0; g < G; g++) {
      const float4 Ui = valid ? Ul[(size_t)g * ncell + cell] : make_float4(0.f, 0.f, 0.f, 0.f);
      const Aux Xi = make_aux(Ui);
      float4 ac = Ui;
      ac.x += dsum[g].x; ac.y += dsum[g].y; ac.z += dsum[g].z; ac.w += dsum[g].w;
#pragma unroll
      for (int a = 0; a < 3; a++) {
        const int bit = (k >> a) & 1;
        const bool sib_leaf = __shfl_xor_sync(0xffffffffu, leaf ? 1 : 0, 1 << a) != 0;
        float4 Us;
        Us.x = __shfl_xor_sync(0xffffffffu, Ui.x, 1 << a); Us.y = __shfl_xor_sync(0xffffffffu, Ui.y, 1 << a);
        Us.z = __shfl_xor_sync(0xffffffffu, Ui.z, 1 << a); Us.w = __shfl_xor_sync(0xffffffffu, Ui.w, 1 << a);
        const AuxD Xa = aux_dir(Xi, a);
        AuxD Xs;                                                       // the sibling's closure and speeds along a, from its lane
        Xs.a = __shfl_xor_sync(0xffffffffu, Xa.a, 1 << a); Xs.b = __shfl_xor_sync(0xffffffffu, Xa.b, 1 << a);
        Xs.lm = __shfl_xor_sync(0xffffffffu, Xa.lm, 1 << a); Xs.lp = __shfl_xor_sync(0xffffffffu, Xa.lp, 1 << a);
        if (leaf && sib_leaf) {
          const float4 d = hll_change(a, 1 - bit, Ui, Xa, Us, Xs, nu);
          ac.x += d.x; ac.y += d.y; ac.z += d.z; ac.w += d.w;
        }
        if (!leaf) continue;
        const int no = nbo[oct * 6 + 2 * a + bit];
        if (no <= -16) {                                               // a coarser leaf: the face's record (amr_ghost_faces_kernel)
          const float4 d = A.dU[l][(size_t)g * A.ucap[l] + 4 * (size_t)(-16 - no) + side_pos(k, a)];
          ac.x += d.x; ac.y += d.y; ac.z += d.z; ac.w += d.w;
          continue;
        }
        float4 Un;
        bool box = false;
        if (no >= 0) {
          const long long nb = ((long long)no << 3) | (k ^ (1 << a));
          if (child && child[nb] >= 0) continue;
          Un = Ul[(size_t)g * ncell + nb];
        } else {
          Un = nb_load(A, box_ghost(-2 - no, a, bit, l, cell), g, Ui);
          box = true;
        }
        const float4 d = hll_change(a, bit, Ui, Xa, Un, make_aux_dir(Un, a), nu);
        ac.x += d.x; ac.y += d.y; ac.z += d.z; ac.w += d.w;
        if (box) acc.outflow -= (double)d.x * dV;
      }
      if (leaf) Unew[(size_t)g * ncell + cell] = ac;
    }
  }
  block_reduce_store(acc, parts + blockIdx.x);
}

// U + sgn G_a(U): what a neighbour on the -(sgn = +1) or +(sgn = -1) side of direction a adds to a cell (the algebra of
// transport.cu: with phi = F/c the update is U' = U (1 - m nu/2) + (nu/2) sum_faces (U_n -/+ G_n) + (nu/2) sum_a p_a G_a(U),
// m = faces that exist, p_a = (- face exists) - (+ face exists); m = 6, p = 0 for a cell with six regular faces)
__device__ __forceinline__ float4 nb_term(const float4& U, float ca, float cb, int a, float sgn)
{
  const float pa = (a == 0) ? U.y : (a == 1) ? U.z : U.w;
  const float u = fmaf(sgn * cb, pa, 1.f);
  float4 r = make_float4(fmaf(sgn, pa, U.x), U.y * u, U.z * u, U.w * u);
  if (a == 0) r.y = fmaf(sgn, ca, r.y); else if (a == 1) r.z = fmaf(sgn, ca, r.z); else r.w = fmaf(sgn, ca, r.w);
  return r;
}

// 8 consecutive lanes hold one oct: across the three sibling faces each lane computes the term its partner needs
// (U +/- G_a of its own state, with its own closure) and the two swap it with shfl.xor by 1, 2, 4: no load and no second
// closure for half of the faces.  The three outer faces go through `nbo` (same-level neighbour oct, derived on the host
// from the paper's neighbour-cell pointers for the static mesh): one dependent load less than nbr -> child.
template <int G>
__global__ void __launch_bounds__(128, AMR_T_CTAS)
amr_transport_kernel(const AmrDev A, int l, float nuh, float4* __restrict__ Unew, double dV, Partial* __restrict__ parts)
{
  Acc acc;
  const long long ncell = A.ncell[l];                                // a multiple of 8
  const float4* __restrict__ Ul = A.U[l];
  const int* __restrict__ child = (l < A.nl) ? A.child[l] : nullptr;
  const int* __restrict__ nbo = A.nbo[l];
  // a level has < 2^31 cells (checked at init): 32-bit cell indices inside a group, one base pointer per group
  const float4* __restrict__ Ug[G];
  float4* __restrict__ Vg[G];
#pragma unroll
  for (int g = 0; g < G; g++) { Ug[g] = Ul + (size_t)g * ncell; Vg[g] = Unew + (size_t)g * ncell; }
  const long long span = (long long)gridDim.x * blockDim.x;
  for (long long base = (long long)blockIdx.x * blockDim.x; base < ncell; base += span) {
    const long long cell = base + threadIdx.x;
    const bool valid = cell < ncell;                                 // uniform per 8-lane group
    const bool leaf = valid && !(child && child[cell] >= 0);
    // only leaves next to a split cell of their own level can have received deposits (bitmap built on the host); the
    // deposit is requested together with the cell's own state so that its latency overlaps with the face work
    const unsigned ci = (unsigned)cell;
    const bool hd = leaf && l < A.nl && ((A.hasdep[l][cell >> 5] >> (cell & 31)) & 1u);
    float4 Ui[G], sum[G], dsum[G];
    float ai[G], bi[G];
    const int k = (int)(cell & 7);
    const long long oct = cell >> 3;
#pragma unroll
    for (int g = 0; g < G; g++) {
      Ui[g] = valid ? Ug[g][ci] : make_float4(0.f, 0.f, 0.f, 0.f);
      sum[g] = make_float4(0.f, 0.f, 0.f, 0.f);
      dsum[g] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll
    for (int g = 0; g < G; g++) closure_ab(Ui[g], ai[g], bi[g]);
    int m = 0;                                                       // faces that exist
    int pmask = 0;                                                   // 2 bits per direction: (- face exists) | (+ face exists) << 1
    // outer faces, indices first (all three pointer loads, then all three split tests, in flight together); a face that
    // does not exist on this level reads the cell itself and is masked out, so the state loads below are branch-free
    int no[3];
    unsigned nb[3];
    bool reg[3];
#pragma unroll
    for (int a = 0; a < 3; a++) no[a] = leaf ? nbo[oct * 6 + 2 * a + ((k >> a) & 1)] : -1;
#pragma unroll
    for (int a = 0; a < 3; a++) nb[a] = (no[a] >= 0) ? (((unsigned)no[a] << 3) | (unsigned)(k ^ (1 << a))) : (valid ? ci : 0u);
    int chn[3];
#pragma unroll
    for (int a = 0; a < 3; a++) chn[a] = (child && no[a] >= 0) ? child[nb[a]] : -1;
#pragma unroll
    for (int a = 0; a < 3; a++) {
      reg[a] = no[a] >= 0 && chn[a] < 0;                             // a leaf of this level behind the face
      if (!reg[a]) nb[a] = valid ? ci : 0u;
    }
#pragma unroll
    for (int a = 0; a < 3; a++) {
      const int bit = (k >> a) & 1;
      // sibling face (side 1 - bit): this lane is the partner's neighbour on side `bit`: it sends U - G (bit = 1) or U + G
      const bool sib_leaf = __shfl_xor_sync(0xffffffffu, leaf ? 1 : 0, 1 << a) != 0;
      const float sg = bit ? -1.f : 1.f;
#pragma unroll
      for (int g = 0; g < G; g++) {
        const float4 T = nb_term(Ui[g], ai[g], bi[g], a, sg);
        const float tx = __shfl_xor_sync(0xffffffffu, T.x, 1 << a), ty = __shfl_xor_sync(0xffffffffu, T.y, 1 << a);
        const float tz = __shfl_xor_sync(0xffffffffu, T.z, 1 << a), tw = __shfl_xor_sync(0xffffffffu, T.w, 1 << a);
        if (sib_leaf) { sum[g].x += tx; sum[g].y += ty; sum[g].z += tz; sum[g].w += tw; }   // split sibling: Fig. 3 (iii)
      }
      if (sib_leaf) { m++; pmask |= 1 << (2 * a + (1 - bit)); }
      // outer face (side = bit): regular neighbour, branch-free
      const float wgt = reg[a] ? 1.f : 0.f;
#pragma unroll
      for (int g = 0; g < G; g++) {
        const float4 Un = Ug[g][nb[a]];
        float an, bn;
        closure_ab(Un, an, bn);
        const float4 T = nb_term(Un, an, bn, a, sg);
        sum[g].x = fmaf(wgt, T.x, sum[g].x); sum[g].y = fmaf(wgt, T.y, sum[g].y);
        sum[g].z = fmaf(wgt, T.z, sum[g].z); sum[g].w = fmaf(wgt, T.w, sum[g].w);
      }
      if (reg[a]) { m++; pmask |= 1 << (2 * a + bit); }
      if (leaf && no[a] <= -2 && no[a] > -16) {                      // box face: -2 - bc (rare: the slow path)
        const NbRef r = box_ghost(-2 - no[a], a, bit, l, cell);
#pragma unroll
        for (int g = 0; g < G; g++) {
          const float4 Un = nb_load(A, r, g, Ui[g]);
          float an, bn;
          closure_ab(Un, an, bn);
          const float4 T = nb_term(Un, an, bn, a, sg);
          sum[g].x += T.x; sum[g].y += T.y; sum[g].z += T.z; sum[g].w += T.w;
          // A15: N-flux through the box face, nu F^ = (nu/2) [(G_i + G_n) -/+ (U_n - U_i)]_N with G_N = phi_a
          const float pi = (a == 0) ? Ui[g].y : (a == 1) ? Ui[g].z : Ui[g].w, pn = (a == 0) ? Un.y : (a == 1) ? Un.z : Un.w;
          const float fl = bit ? nuh * ((pi + pn) - (Un.x - Ui[g].x)) : -nuh * ((pi + pn) - (Ui[g].x - Un.x));
          acc.outflow += (double)fl * dV;
        }
        m++; pmask |= 1 << (2 * a + bit);
      }
    }
    if (!leaf) continue;
    const float own = fmaf(-nuh, (float)m, 1.f);
    float4 ac[G];
#pragma unroll
    for (int g = 0; g < G; g++) {
      ac[g].x = fmaf(nuh, sum[g].x, own * Ui[g].x); ac[g].y = fmaf(nuh, sum[g].y, own * Ui[g].y);
      ac[g].z = fmaf(nuh, sum[g].z, own * Ui[g].z); ac[g].w = fmaf(nuh, sum[g].w, own * Ui[g].w);
    }
    if (pmask != 63) {                                               // a missing face: the own flux does not cancel
#pragma unroll
      for (int a = 0; a < 3; a++) {
        const int p = ((pmask >> (2 * a)) & 1) - ((pmask >> (2 * a + 1)) & 1);
        if (p == 0) continue;
#pragma unroll
        for (int g = 0; g < G; g++) {
          const float4 Gv = flux_vec(Ui[g], ai[g], bi[g], a);
          const float w = nuh * (float)p;
          ac[g].x = fmaf(w, Gv.x, ac[g].x); ac[g].y = fmaf(w, Gv.y, ac[g].y);
          ac[g].z = fmaf(w, Gv.z, ac[g].z); ac[g].w = fmaf(w, Gv.w, ac[g].w);
        }
      }
    }
    // the finer level's deposits (gathered here, after the regular faces: only few cells have any, and their dependent loads
    // must not sit in front of everyone's neighbour loads), then the faces towards a coarser leaf (records of
    // amr_ghost_faces_kernel), x, y, z: a fixed order of plain additions -- no other thread touches this cell
    if (hd) {                                                        // gather the finer level's deposits (few cells)
#pragma unroll
      for (int a = 0; a < 3; a++) {
        const int bit = (k >> a) & 1;
        const int chs = child[cell ^ (1 << a)];                      // the sibling across a (same oct record)
        if (chs >= 0) gather_side<G>(A, l, chs, 2 * a + (1 - bit), dsum);
        if (chn[a] >= 0) gather_side<G>(A, l, chn[a], 2 * a + bit, dsum);
      }
    }

#pragma unroll
    for (int g = 0; g < G; g++) { ac[g].x += dsum[g].x; ac[g].y += dsum[g].y; ac[g].z += dsum[g].z; ac[g].w += dsum[g].w; }
#pragma unroll
    for (int a = 0; a < 3; a++)
      if (no[a] <= -16) {
        const size_t rec = 4 * (size_t)(-16 - no[a]) + side_pos(k, a);
#pragma unroll
        for (int g = 0; g < G; g++) {
          const float4 d = A.dU[l][(size_t)g * A.ucap[l] + rec];
          ac[g].x += d.x; ac[g].y += d.y; ac[g].z += d.z; ac[g].w += d.w;
        }
      }
#pragma unroll
    for (int g = 0; g < G; g++) Vg[g][ci] = ac[g];
  }
  block_reduce_store(acc, parts + blockIdx.x);
}

// The faces of refined leaves that look at a coarser leaf (resolution jump), one thread per face from a list the host
// built once for the static mesh: the six coarse references are resolved once, then per group the MinMod ghost
// (PAPER.md:436), the Eq. 32 flux, the fine cell's change (a record the per-cell kernel adds to its result) and the same
// flux / 8 for the coarse leaf (Fig. 3 (i)-(ii); a record per oct side that the leaf gathers).  Uniform work per thread: the irregular part of the
// level is taken out of the per-cell kernel, where it made every warp on a patch boundary run the ghost code.
template <int G, bool HLL>
__global__ void __launch_bounds__(128)
amr_ghost_faces_kernel(const AmrDev A, int l, float nuh, int sub, const int* __restrict__ slot_cell,
                       const int* __restrict__ slot_coarse, const unsigned char* __restrict__ slot_face,
                       const int* __restrict__ slot_refs, int n_slots)
{
  const int i0 = blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = i0 < n_slots;                                   // n_slots is a multiple of 4: uniform per 4 lanes
  const int i = live ? i0 : n_slots - 1;                            // idle lanes redo the last entry, write nothing
  const long long cell = slot_cell[i], c = slot_coarse[i];
  const int f = slot_face[i], a = f >> 1, side = f & 1, lc = l - 1;
  const int kv = (int)(cell & 7) ^ (1 << a);                        // child index of the virtual cell inside c
  const long long ncell = A.ncell[l], ncc = A.ncell[lc];
  // the six level-(l-1) neighbours of c, resolved on the host for the static mesh (one record per oct side):
  //   >= 0 a cell of level l-1; <= -16 the coarser leaf -16 - code of level l-2 (piecewise constant); -1 box ghost = c
  //   itself; -2, -3, -4 the same with flux component 0, 1, 2 inverted (A13); -5 the inflow state of that face (A20)
  int rc[6];
#pragma unroll
  for (int j = 0; j < 6; j++) rc[j] = slot_refs[(size_t)(i >> 2) * 6 + j];
  const long long ncc2 = lc > 0 ? A.ncell[lc - 1] : 0;
#pragma unroll
  for (int g = 0; g < G; g++) {
    const float4 Uc = A.U[lc][(size_t)g * ncc + c];
    float4 Unb[6];
#pragma unroll
    for (int j = 0; j < 6; j++) {
      const int code = rc[j];
      if (code >= 0) Unb[j] = A.U[lc][(size_t)g * ncc + code];
      else if (code <= -16) Unb[j] = A.U[lc - 1][(size_t)g * ncc2 + (-16 - code)];
      else if (code == -5) Unb[j] = A.inflow[j][g];
      else {
        Unb[j] = Uc;
        if (code == -2) Unb[j].y = -Uc.y; else if (code == -3) Unb[j].z = -Uc.z; else if (code == -4) Unb[j].w = -Uc.w;
      }
    }
    float4 Un = Uc;
#pragma unroll
    for (int b = 0; b < 3; b++) {
      const float4 Um = Unb[2 * b], Up = Unb[2 * b + 1];
      const float sg = ((kv >> b) & 1) ? 0.25f : -0.25f;
      Un.x = fmaf(sg, minmod(Uc.x - Um.x, Up.x - Uc.x), Un.x);
      Un.y = fmaf(sg, minmod(Uc.y - Um.y, Up.y - Uc.y), Un.y);
      Un.z = fmaf(sg, minmod(Uc.z - Um.z, Up.z - Uc.z), Un.z);
      Un.w = fmaf(sg, minmod(Uc.w - Um.w, Up.w - Uc.w), Un.w);
    }
    const float4 Ui = A.U[l][(size_t)g * ncell + cell];
    float4 d;
    if (HLL) d = hll_change(a, side, Ui, make_aux_dir(Ui, a), Un, make_aux_dir(Un, a), 2.f * nuh);
    else {
      float ai, bi;
      closure_ab(Ui, ai, bi);
      d = face_change(a, side, Ui, ai, bi, Un, nuh);
    }
    if (live) A.dU[l][(size_t)g * A.ucap[l] + i] = d;               // read by the cell kernel of this level, this sweep
    // the 4 faces of one oct side are 4 consecutive list entries (aligned lanes) and share the coarse leaf: one deposit
    float4 s4 = d;
    s4.x += __shfl_xor_sync(0xffffffffu, s4.x, 1); s4.y += __shfl_xor_sync(0xffffffffu, s4.y, 1);
    s4.z += __shfl_xor_sync(0xffffffffu, s4.z, 1); s4.w += __shfl_xor_sync(0xffffffffu, s4.w, 1);
    s4.x += __shfl_xor_sync(0xffffffffu, s4.x, 2); s4.y += __shfl_xor_sync(0xffffffffu, s4.y, 2);
    s4.z += __shfl_xor_sync(0xffffffffu, s4.z, 2); s4.w += __shfl_xor_sync(0xffffffffu, s4.w, 2);
    if ((threadIdx.x & 3) == 0 && live) {                             // gathered by the coarse leaf when its own step comes
      float4* rp = A.depS[l] + (size_t)g * A.scap[l] + (size_t)(cell >> 3) * 6 + f;
      float4 r = make_float4(-0.125f * s4.x, -0.125f * s4.y, -0.125f * s4.z, -0.125f * s4.w);
      if (sub) { const float4 o = *rp; r.x += o.x; r.y += o.y; r.z += o.z; r.w += o.w; }   // second sub-step: first + second
      *rp = r;
    }
  }
}

// Eq. 43-48 on the leaves of a refined level, in place, over cp.dt (= dt / 2^level)
template <int G>
__global__ void __launch_bounds__(128, 8)
amr_chem_kernel(const ChemParams cp, const LevelDev L, float4* __restrict__ U, const int* __restrict__ child,
                int count_total, int limit, Partial* __restrict__ parts)
{
  Acc acc;
  const long long ncell = L.ncell;
  for (long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x; cell < ncell; cell += (long long)gridDim.x * blockDim.x) {
    if (child && child[cell] >= 0) { if (cp.record) L.subc[cell] = 0; continue; }
    CellState<G> c;
    load_cell<G>(L, cell, U, ncell, cell, c);
    if (limit) {                                                      // HLL (A19): the transported state is made realizable
#pragma unroll
      for (int g = 0; g < G; g++) {
        float4 u = make_float4(c.N[g], c.px[g], c.py[g], c.pz[g]);
        realizable(u);
        c.px[g] = u.y; c.py[g] = u.z; c.pz[g] = u.w;
      }
    }
    CellTally tl;
    float rem = cp.dt, dmin = FINF;
    bool ok = true;
    while (ok && rem > 0.f) ok = substep<G>(cp, c, rem, tl, dmin);
    if (!ok) acc.err |= 1u;
    store_cell<G>(L, cell, U, ncell, c, tl, cp.record);
    const double before = acc.total;
    fold(acc, tl, c.N, G, L.dV, L.dV_total);
    if (!count_total) acc.total = before;                            // photons are counted once per coarse step
    acc.dtau_min = fminf(acc.dtau_min, dmin);
    if (!finite_cell<G>(c)) acc.nonfinite++;
  }
  block_reduce_store(acc, parts + blockIdx.x);
}

// chemistry off (A9): N += S dt in the source cells of the level; count_total: also sum N dV over the leaves
template <int G>
__global__ void __launch_bounds__(128)
amr_sources_kernel(const LevelDev L, float4* __restrict__ U, const int* __restrict__ child, float dt, int count_total,
                   int limit, Partial* __restrict__ parts)
{
  Acc acc;
  const long long ncell = L.ncell;
  for (long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x; cell < ncell; cell += (long long)gridDim.x * blockDim.x) {
    if (child && child[cell] >= 0) continue;
    float S[G];
    load_sources<G>(L, cell, S);
    float s = 0.f;
#pragma unroll
    for (int g = 0; g < G; g++) {
      float4* p = U + (size_t)g * ncell + cell;
      if (limit) { float4 u = *p; realizable(u); *p = u; }          // HLL (A19)
      if (S[g] != 0.f) {
        const float add = S[g] * dt;
        p->x += add;
        acc.injected += (double)add * L.dV;
      }
      s += p->x;
    }
    if (count_total) acc.total += (double)s * L.dV;
  }
  block_reduce_store(acc, parts + blockIdx.x);
}

__device__ __forceinline__ float oct_sum8(float v)
{
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  v += __shfl_xor_sync(0xffffffffu, v, 4);
  return v;
}

// split cell := mean of its 8 children (N, phi; with_gas: x and e too), 8 lanes per oct
template <int G>
__global__ void __launch_bounds__(256)
amr_restrict_kernel(const LevelDev L, const LevelDev Lbelow, const float4* __restrict__ Uf, float4* __restrict__ Uc,
                    int with_gas)
{
  const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = cell < L.ncell;                                  // uniform per 8-lane group
  float4 m[G];
#pragma unroll
  for (int g = 0; g < G; g++) {
    const float4 u = valid ? Uf[(size_t)g * L.ncell + cell] : make_float4(0.f, 0.f, 0.f, 0.f);
    m[g].x = 0.125f * oct_sum8(u.x); m[g].y = 0.125f * oct_sum8(u.y);
    m[g].z = 0.125f * oct_sum8(u.z); m[g].w = 0.125f * oct_sum8(u.w);
  }
  float x = 0.f, y = 0.f, e = 0.f;
  if (valid && with_gas) { decode_x(L.xs[cell], x, y); e = L.eps[cell] * L.n0[cell]; }
  const float xm = 0.125f * oct_sum8(x), ym = 0.125f * oct_sum8(y), em = 0.125f * oct_sum8(e);
  if (valid && (cell & 7) == 0) {
    const long long pc = L.parent[cell >> 3];
#pragma unroll
    for (int g = 0; g < G; g++) Uc[(size_t)g * Lbelow.ncell + pc] = m[g];
    if (with_gas) { Lbelow.xs[pc] = encode_x(xm, ym); Lbelow.eps[pc] = em / Lbelow.n0[pc]; }
  }
}

// refined cells start with the radiation of their parent
template <int G>
__global__ void amr_inject_init_kernel(const LevelDev L, const float4* __restrict__ Uc, long long ncell_c, float4* __restrict__ Uf)
{
  const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cell >= L.ncell) return;
  const long long pc = L.parent[cell >> 3];
#pragma unroll
  for (int g = 0; g < G; g++) Uf[(size_t)g * L.ncell + cell] = Uc[(size_t)g * ncell_c + pc];
}

// level 0 after the dense pass: the leaves with a split face neighbour are recomputed from the old states, face by
// face, without the faces that look at a split cell (Fig. 3 (iii)), plus what the fine cells behind those faces
// deposited during their two sub-steps.  Recomputed, not corrected: taking a large coarse flux back out of the dense
// result would leave its rounding error on a possibly much smaller remainder.
template <int G, bool HLL>
__global__ void __launch_bounds__(128)
amr_fix0_kernel(const AmrDev A, const float4* __restrict__ Uold, float4* __restrict__ Unew, const int* __restrict__ fix_cell,
                const unsigned char* __restrict__ fix_mask, int n_fix, float nuh)
{
  const int t = blockIdx.x * blockDim.x + threadIdx.x;                // one thread per (cell, group): independent loads
  if (t >= n_fix * G) return;
  const int i = t / G, g = t - i * G;
  const long long cell = fix_cell[i];
  const unsigned mask = fix_mask[i];
  const long long nc = A.ncell[0];
  // all seven states and the deposit are requested before anything is used (the cells are scattered: one DRAM round
  // trip instead of seven); a masked or box face reads the cell itself
  const int n = A.n;
  const unsigned uc = (unsigned)cell, tq = uc / (unsigned)n;
  const int ci[3] = {(int)(uc % (unsigned)n), (int)(tq % (unsigned)n), (int)(tq / (unsigned)n)};
  const long long stride[3] = {1, n, (long long)n * n};
  long long idx[6];
  int ghost[6];                                                     // 0 cell, 1 transmissive, 2 reflective, 3 inflow
  bool on[6];
#pragma unroll
  for (int f = 0; f < 6; f++) {
    const int a = f >> 1, side = f & 1, cn = ci[a] + (side ? 1 : -1);
    on[f] = !((mask >> f) & 1u);
    ghost[f] = 0;
    idx[f] = cell + (side ? stride[a] : -stride[a]);
    if (cn < 0 || cn >= n) {
      const int bc = A.bc[f];
      if (bc == EMMA_RT_BC_PERIODIC) idx[f] = cell + (side ? -(long long)(n - 1) : (long long)(n - 1)) * stride[a];
      else { idx[f] = cell; ghost[f] = bc; }
    }
  }
  // what the fine cells behind the split neighbours handed to this leaf (Fig. 3 (i)-(ii)): the records of the two sub-steps
  // of level 1, face by face in a fixed order
  float4 dpv = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
  for (int f = 0; f < 6; f++)
    if (!on[f]) {
      const int o2 = A.child[0][idx[f]];
      const size_t sd = (size_t)o2 * 6 + (f ^ 1);
      const float4 r = A.depS[1][(size_t)g * A.scap[1] + sd];
      dpv.x += r.x; dpv.y += r.y; dpv.z += r.z; dpv.w += r.w;
      idx[f] = cell;
    }
  const float4 Ui = Uold[(size_t)g * nc + cell];
  float4 Un[6];
#pragma unroll
  for (int f = 0; f < 6; f++) Un[f] = Uold[(size_t)g * nc + idx[f]];
#pragma unroll
  for (int f = 0; f < 6; f++) {
    if (ghost[f] == EMMA_RT_BC_INFLOW) Un[f] = A.inflow[f][g];
    else if (ghost[f] == EMMA_RT_BC_REFLECTIVE) { if ((f >> 1) == 0) Un[f].y = -Un[f].y; else if ((f >> 1) == 1) Un[f].z = -Un[f].z; else Un[f].w = -Un[f].w; }
  }
  float4 ac = Ui;
  if (HLL) {
    const Aux Xi = make_aux(Ui);
#pragma unroll
    for (int f = 0; f < 6; f++)
      if (on[f]) {
        const float4 d = hll_change(f >> 1, f & 1, Ui, aux_dir(Xi, f >> 1), Un[f], make_aux_dir(Un[f], f >> 1), 2.f * nuh);
        ac.x += d.x; ac.y += d.y; ac.z += d.z; ac.w += d.w;
      }
  } else {
    float ai, bi;
    closure_ab(Ui, ai, bi);
#pragma unroll
    for (int f = 0; f < 6; f++)
      if (on[f]) {
        const float4 d = face_change(f >> 1, f & 1, Ui, ai, bi, Un[f], nuh);
        ac.x += d.x; ac.y += d.y; ac.z += d.z; ac.w += d.w;
      }
  }
  ac.x += dpv.x; ac.y += dpv.y; ac.z += dpv.z; ac.w += dpv.w;
  if (HLL) realizable(ac);                                            // A19, after the deposits
  Unew[(size_t)g * nc + cell] = ac;
}

// net N-flux through the non-periodic box faces of the level-0 LEAVES (the dense pass also counts split cells, whose
// faces belong to their children here), from the old states
template <int G, bool HLL>
__global__ void __launch_bounds__(128)
amr_outflow0_kernel(const AmrDev A, const float4* __restrict__ Uold, float nuh, double dV, Partial* __restrict__ parts)
{
  Acc acc;
  const int n = A.n;
  const long long per = (long long)n * n, nc = A.ncell[0];
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < 6 * per; t += (long long)gridDim.x * blockDim.x) {
    const int f = (int)(t / per), a = f >> 1, side = f & 1;
    if (A.bc[f] == EMMA_RT_BC_PERIODIC) continue;
    const int u = (int)(t % n), v = (int)((t / n) % n), w = side ? n - 1 : 0;
    const long long cell = (a == 0) ? w + (long long)n * (u + (long long)n * v)
                         : (a == 1) ? u + (long long)n * (w + (long long)n * v) : u + (long long)n * (v + (long long)n * w);
    if (A.child[0] && A.child[0][cell] >= 0) continue;
    const NbRef r = nb_ref0(A, cell, a, side);
#pragma unroll
    for (int g = 0; g < G; g++) {
      const float4 Ui = Uold[(size_t)g * nc + cell];
      const float4 Un = nb_load(A, r, g, Ui);
      float4 d;
      if (HLL) d = hll_change(a, side, Ui, make_aux_dir(Ui, a), Un, make_aux_dir(Un, a), 2.f * nuh);
      else {
        float ai, bi;
        closure_ab(Ui, ai, bi);
        d = face_change(a, side, Ui, ai, bi, Un, nuh);
      }
      acc.outflow -= (double)d.x * dV;
    }
  }
  block_reduce_store(acc, parts + blockIdx.x);
}

int grid_for(long long work, int block, int cap)
{
  long long b = (work + block - 1) / block;
  if (b < 1) b = 1;
  if (b > cap) b = cap;
  return (int)b;
}
constexpr int AMR_GRID_CAP = 148 * 8;            // (the transport kernel uses 148 * AMR_T_CTAS)            // whole waves of 8 CTAs of 128 threads per SM; each block writes one Partial

}  // namespace

#define AMR_DISPATCH(G, CALL)                                   \
  switch (G) {                                                  \
    case 1: { constexpr int GG = 1; CALL; } break;              \
    case 2: { constexpr int GG = 2; CALL; } break;              \
    case 3: { constexpr int GG = 3; CALL; } break;              \
    default: { constexpr int GG = 4; CALL; } break;             \
  }

int launch_amr_transport(const AmrDev& A, int level, float nuh, float4* Unew, double dV, int hll, Partial* parts, int* n_parts,
                         cudaStream_t st)
{
  const int nb = grid_for(A.ncell[level], 128, 148 * AMR_T_CTAS);
  if (hll) { AMR_DISPATCH(A.G, (amr_transport_hll_kernel<GG><<<nb, 128, 0, st>>>(A, level, nuh, Unew, dV, parts))); }
  else AMR_DISPATCH(A.G, (amr_transport_kernel<GG><<<nb, 128, 0, st>>>(A, level, nuh, Unew, dV, parts)));
  *n_parts = nb;
  return 1;
}

int launch_amr_ghost_faces(const AmrDev& A, int level, float nuh, int sub, const int* slot_cell, const int* slot_coarse,
                           const unsigned char* slot_face, const int* slot_refs, int n_slots, int hll, cudaStream_t st)
{
  if (n_slots == 0) return 0;
  const int nb = (n_slots + 127) / 128;
  if (hll) { AMR_DISPATCH(A.G, (amr_ghost_faces_kernel<GG, true><<<nb, 128, 0, st>>>(A, level, nuh, sub, slot_cell, slot_coarse, slot_face, slot_refs, n_slots))); }
  else AMR_DISPATCH(A.G, (amr_ghost_faces_kernel<GG, false><<<nb, 128, 0, st>>>(A, level, nuh, sub, slot_cell, slot_coarse, slot_face, slot_refs, n_slots)));
  return 1;
}

int launch_amr_chem(const ChemParams& cp, const LevelDev& L, const AmrDev& A, int level, int count_total, int limit,
                    Partial* parts, int* n_parts, cudaStream_t st)
{
  const int nb = grid_for(L.ncell, 128, AMR_GRID_CAP);
  const int* child = level < A.nl ? A.child[level] : nullptr;
  AMR_DISPATCH(A.G, (amr_chem_kernel<GG><<<nb, 128, 0, st>>>(cp, L, A.U[level], child, count_total, limit, parts)));
  *n_parts = nb;
  return 1;
}

int launch_amr_sources(const LevelDev& L, const AmrDev& A, int level, float dt, int count_total, int limit, Partial* parts,
                       int* n_parts, cudaStream_t st)
{
  const int nb = grid_for(L.ncell, 128, AMR_GRID_CAP);
  const int* child = level < A.nl ? A.child[level] : nullptr;
  AMR_DISPATCH(A.G, (amr_sources_kernel<GG><<<nb, 128, 0, st>>>(L, A.U[level], child, dt, count_total, limit, parts)));
  *n_parts = nb;
  return 1;
}

int launch_amr_restrict(const LevelDev& Lfine, const LevelDev& Lcoarse, const AmrDev& A, int level_fine, int with_gas,
                        cudaStream_t st)
{
  if (Lfine.ncell == 0) return 0;
  const int nb = (int)((Lfine.ncell + 255) / 256);
  AMR_DISPATCH(A.G, (amr_restrict_kernel<GG><<<nb, 256, 0, st>>>(Lfine, Lcoarse, A.U[level_fine], A.U[level_fine - 1], with_gas)));
  return 1;
}

int launch_amr_inject_init(const LevelDev& Lfine, const AmrDev& A, int level_fine, cudaStream_t st)
{
  if (Lfine.ncell == 0) return 0;
  const int nb = (int)((Lfine.ncell + 255) / 256);
  AMR_DISPATCH(A.G, (amr_inject_init_kernel<GG><<<nb, 256, 0, st>>>(Lfine, A.U[level_fine - 1], A.ncell[level_fine - 1], A.U[level_fine])));
  return 1;
}

int launch_amr_fix0(const AmrDev& A, const float4* Uold, float4* Unew, const int* fix_cell, const unsigned char* fix_mask,
                    int n_fix, float nuh, int hll, cudaStream_t st)
{
  if (n_fix == 0) return 0;
  const int nb = (int)(((long long)n_fix * A.G + 127) / 128);
  if (hll) { AMR_DISPATCH(A.G, (amr_fix0_kernel<GG, true><<<nb, 128, 0, st>>>(A, Uold, Unew, fix_cell, fix_mask, n_fix, nuh))); }
  else AMR_DISPATCH(A.G, (amr_fix0_kernel<GG, false><<<nb, 128, 0, st>>>(A, Uold, Unew, fix_cell, fix_mask, n_fix, nuh)));
  return 1;
}

int launch_amr_outflow0(const AmrDev& A, const float4* Uold, float nuh, double dV, int hll, Partial* parts, int* n_parts,
                        cudaStream_t st)
{
  const int nb = grid_for(6LL * A.n * A.n, 128, 148 * 2);
  if (hll) { AMR_DISPATCH(A.G, (amr_outflow0_kernel<GG, true><<<nb, 128, 0, st>>>(A, Uold, nuh, dV, parts))); }
  else AMR_DISPATCH(A.G, (amr_outflow0_kernel<GG, false><<<nb, 128, 0, st>>>(A, Uold, nuh, dV, parts)));
  *n_parts = nb;
  return 1;
}

}  // namespace emma
