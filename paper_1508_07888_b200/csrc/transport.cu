// transport.cu -- explicit M1 transport on the coarse block.
//
// U = (N, F), flux F~ = (F, c^2 P), Eq. 30 (conservative update) with the Lax-Friedrichs /
// GLF interface flux Eq. 32, unsplit over the three directions (A4), closure Eq. 22-23 (A1, A2), reduced speed
// of light everywhere (A3), boundary conditions of PAPER.md:436 (A13).
//
// In the internal variables phi = F / c the own-cell flux cancels and the whole update is
//     U' = (1 - 3 nu) U + (nu/2) sum_d [ (U - G_d)(i+e_d) + (U + G_d)(i-e_d) ],     nu = c dt / dx,
//     G_d = (phi_d, Pi_dx, Pi_dy, Pi_dz),   Pi = P (in units of N) = a I + b phi(x)phi,
//     a = N (1/3 - q),  b = 3 q / (N f^2),  q = f^2 / (2 + sqrt(4 - 3 f^2)),  f = |phi| / N clipped to 1
// (algebraically Levermore's chi = 1/3 + 2q; the form avoids the cancellation of 3 chi - 1 at small f).
// Each cell's closure (a, b) is computed ONCE, by the thread that owns the cell (or its halo copy), and staged in
// shared memory next to U; the paper's own stencil-array design recomputes it for every neighbour.
//
// Kernel shape: 2.5-D streaming.  A CTA owns a TX x TY column of cells and marches along z through a chunk of
// planes; every thread owns CY = 2 cells adjacent in y.  z-neighbours (and the y-neighbour inside the pair) live in
// registers, the other x/y-neighbours come from a double-buffered shared-memory plane (one barrier per plane).
// Loads of plane k+2 are issued while plane k is computed.  HBM traffic is the algorithmic 16 B read + 16 B write
// per cell-group plus the tile-edge halo (served from L2).
//
// The first version of this kernel was issue-bound (ncu: 82 % issue slots busy, 291 instructions per cell-group,
// profiles/r1a_*): this one is written for instruction count -- packed fp32 (FFMA2 on the (N,phi_x) and
// (phi_y,phi_z) register pairs of the float4), pointer increments instead of 64-bit index arithmetic, diagnostics
// compiled in only where a configuration needs them.
#include "emma_rt_internal.cuh"
#include "transport_math.cuh"

namespace emma {

namespace {

constexpr int TX = 32;                         // tile width = one warp along x
constexpr int TYT = 8;                         // thread rows
constexpr int CY = 2;                          // cells per thread along y
constexpr int TY = TYT * CY;
constexpr int NT = TX * TYT;
constexpr int SW = TX + 2;                     // shared plane width incl. halo
constexpr int SH = TY + 2;

// One plane of the z pipeline held in registers: my two cells (raw U and closure) and my halo cell.
struct Slot {
  float4 u0, u1, h;
  float a0, b0, a1, b1;
};

struct Tile {                                  // per-thread constants of the march
  int tx, ly, hsx, hsy;
  bool act0, act1, pair, hduty;
  float hsgn_y, hsgn_z;
};

// DIAG: chemistry is off, so this pass owns the step's photon total and non-finite scan.
// OPEN: some face is transmissive or an inflow face (A20), so the pass sums the outflow of A15 (and inflow ghosts exist).
template <bool DIAG, bool OPEN>
__global__ void __launch_bounds__(NT, 2)
transport_kernel(const TransportParams p, const float4* __restrict__ Uin, float4* __restrict__ Uout,
                 Partial* __restrict__ parts)
{
  __shared__ float4 sU[3][SH][SW];
  __shared__ float2 sAB[3][SH][SW];

  const int n = p.n;
  // block -> (tile x, tile y, z chunk, group), tile x fastest so that concurrently resident CTAs are neighbours
  int bid = blockIdx.x;
  const int tix = bid % p.tiles_x; bid /= p.tiles_x;
  const int tiy = bid % p.tiles_y; bid /= p.tiles_y;
  const int izc = bid % p.nzc;     bid /= p.nzc;
  const int g = bid;
  const int x0 = tix * TX, y0 = tiy * TY;
  const int wx = min(TX, n - x0), wy = min(TY, n - y0);
  const int z0 = izc * p.zchunk, z1 = min(n, z0 + p.zchunk);
  Tile T;
  T.tx = threadIdx.x % TX;
  T.ly = CY * (threadIdx.x / TX);              // first of my two rows inside the tile
  T.pair = T.ly + 1 < wy;                      // warp-uniform: both of my rows are inside the tile
  T.act0 = (T.tx < wx) && (T.ly < wy);
  T.act1 = (T.tx < wx) && T.pair;
  const int x = x0 + T.tx, y = y0 + T.ly;
  const size_t plane = (size_t)n * n;
  const float4* __restrict__ Ug = Uin + (size_t)g * plane * n;
  const size_t col0 = T.act0 ? ((size_t)y * n + x) : 0;
  const size_t col1 = T.act1 ? col0 + n : col0;

  // halo duty: thread t < 2*wy + 2*wx also stages one halo cell per plane
  const int t = threadIdx.x;
  T.hduty = t < 2 * wy + 2 * wx;
  T.hsx = 0; T.hsy = 0;
  int hflipc = 0;                              // component of the halo cell to flip (1..2) or 0
  size_t hcol = 0;
  if (T.hduty) {
    bool fl;
    if (t < 2 * wy) {                          // left / right columns
      const int r = (t < wy) ? t : t - wy;
      const int gx = bc_map((t < wy) ? x0 - 1 : x0 + wx, n, p.bc[0], p.bc[1], fl);
      T.hsx = (t < wy) ? 0 : wx + 1; T.hsy = r + 1;
      hcol = (size_t)(y0 + r) * n + gx;
      hflipc = fl ? 1 : 0;
    } else {                                   // bottom / top rows
      const int q = t - 2 * wy;
      const int r = (q < wx) ? q : q - wx;
      const int gy = bc_map((q < wx) ? y0 - 1 : y0 + wy, n, p.bc[2], p.bc[3], fl);
      T.hsx = r + 1; T.hsy = (q < wx) ? 0 : wy + 1;
      hcol = (size_t)gy * n + (x0 + r);
      hflipc = fl ? 2 : 0;
    }
  }
  T.hsgn_y = (hflipc == 1) ? -1.f : 1.f;
  T.hsgn_z = (hflipc == 2) ? -1.f : 1.f;
  // inflow faces (A20): the ghost is a prescribed state, not a cell of the grid
  bool hin = false;
  float4 hval = make_float4(0.f, 0.f, 0.f, 0.f);
  if (OPEN && T.hduty) {
    int face = -1;
    if (t < wy) { if (x0 == 0) face = 0; }
    else if (t < 2 * wy) { if (x0 + wx == n) face = 1; }
    else if (t - 2 * wy < wx) { if (y0 == 0) face = 2; }
    else { if (y0 + wy == n) face = 3; }
    if (face >= 0 && p.bc[face] == EMMA_RT_BC_INFLOW) { hin = true; hval = p.inflow[face][g]; }
  }
  const bool zin_lo = OPEN && z0 == 0 && p.bc[4] == EMMA_RT_BC_INFLOW;
  const bool zin_hi = OPEN && z1 == n && p.bc[5] == EMMA_RT_BC_INFLOW;

  const int pfd = p.pf;
  const float c0 = p.c0, c1 = p.c1;
  Acc acc_d;

  // ---- prologue: planes z0-1 (-> W), z0 (-> slot A), z0+1 (-> slot B, raw); halo of z0, z0+1
  bool flz, fltop;
  const int zm = bc_map(z0 - 1, n, p.bc[4], p.bc[5], flz);
  const int ztop = bc_map(z1, n, p.bc[4], p.bc[5], fltop);      // the plane above the chunk (mapped)
  const float sgtop = fltop ? -1.f : 1.f;
  const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
  Slot A, B, C;
  A.u0 = A.u1 = A.h = B.u0 = B.u1 = B.h = C.u0 = C.u1 = C.h = zero4;
  A.a0 = A.b0 = A.a1 = A.b1 = B.a0 = B.b0 = B.a1 = B.b1 = C.a0 = C.b0 = C.a1 = C.b1 = 0.f;
  float4 W0, W1;
  {
    const float4* pm = Ug + (size_t)zm * plane;
    const float4* pc = Ug + (size_t)z0 * plane;
    const float4* pn = Ug + (size_t)((z0 + 1 < z1) ? z0 + 1 : ztop) * plane;
    float4 m0 = zero4, m1 = zero4;
    if (T.act0) { m0 = __ldg(pm + col0); A.u0 = __ldg(pc + col0); B.u0 = __ldg(pn + col0); }
    if (T.act1) { m1 = __ldg(pm + col1); A.u1 = __ldg(pc + col1); B.u1 = __ldg(pn + col1); }
    if (T.hduty) {
      A.h = hin ? hval : __ldg(pc + hcol);
      if (z0 + 1 < z1) B.h = hin ? hval : __ldg(pn + hcol);
    }
    if (zin_lo) m0 = m1 = p.inflow[4][g];
    if (zin_hi && z0 + 1 >= z1) B.u0 = B.u1 = p.inflow[5][g];
    if (flz) { m0.w = -m0.w; m1.w = -m1.w; }
    float a, b;
    closure_ab(m0, a, b); W0 = below_z(m0, a, b);
    closure_ab(m1, a, b); W1 = below_z(m1, a, b);
    closure_ab(A.u0, A.a0, A.b0);
    closure_ab(A.u1, A.a1, A.b1);
  }
  // running pointers (own column 0): loads of plane z+2, stores of plane z
  const float4* pld = Ug + (size_t)(z0 + 2) * plane + col0;
  const float4* ptop = Ug + (size_t)ztop * plane + col0;
  float4* pst = Uout + (size_t)g * plane * n + (size_t)z0 * plane + col0;
  const ptrdiff_t d1 = (ptrdiff_t)(col1 - col0), dh = (ptrdiff_t)hcol - (ptrdiff_t)col0;
  float sg_nxt = (z0 + 1 == z1) ? sgtop : 1.f;                  // sign of phi_z of the plane held in the next slot
  int z = z0;

  // one plane: CUR is staged and updated, NXT (already loaded) gets its closure, NEW receives the loads of z+2
  auto body = [&](Slot& CUR, Slot& NXT, Slot& NEW, const int buf) {
    // (a) stage this plane: own cells and halo cell, each with its closure
    if (T.act0) { sU[buf][T.ly + 1][T.tx + 1] = CUR.u0; sAB[buf][T.ly + 1][T.tx + 1] = make_float2(CUR.a0, CUR.b0); }
    if (T.act1) { sU[buf][T.ly + 2][T.tx + 1] = CUR.u1; sAB[buf][T.ly + 2][T.tx + 1] = make_float2(CUR.a1, CUR.b1); }
    if (T.hduty) {
      float4 h = CUR.h;
      h.y *= T.hsgn_y; h.z *= T.hsgn_z;
      float a, b;
      closure_ab(h, a, b);
      sU[buf][T.hsy][T.hsx] = h;
      sAB[buf][T.hsy][T.hsx] = make_float2(a, b);
    }
    // (b) issue the loads of plane z+2 (consumed one iteration from now)
    const bool last2 = (z + 2 >= z1);                           // plane z+2 is the (mapped) plane above the chunk
    if (z + 1 < z1) {
      const float4* q = last2 ? ptop : pld;
      if (T.act0) NEW.u0 = __ldg(q);
      if (T.act1) NEW.u1 = __ldg(q + d1);
      if (last2 && zin_hi) NEW.u0 = NEW.u1 = p.inflow[5][g];
      if (T.hduty && !last2) NEW.h = hin ? hval : __ldg(q + dh);
    }
    // (b') L2 prefetch of plane z+2+pfd: own cells and the halo cell (the halo columns are 32 separate sectors per
    // warp load, the slowest request of the plane).  Measured at 512^3 x 3: 4.19 -> 4.64 TB/s.
    if (pfd > 0 && z + 2 + pfd < z1) {
      const float4* q = pld + (size_t)pfd * plane;
      if (T.act0) prefetch_l2(q);
      if (T.act1) prefetch_l2(q + d1);
      if (T.hduty) prefetch_l2(q + dh);
    }
    // (c) closure of the plane above and its contribution U - G_z
    float4 acc0 = W0, acc1 = W1;
    NXT.u0.w *= sg_nxt; NXT.u1.w *= sg_nxt;
    closure_ab(NXT.u0, NXT.a0, NXT.b0);
    closure_ab(NXT.u1, NXT.a1, NXT.b1);
    add_plus<2>(acc0, NXT.u0, NXT.a0, NXT.b0);
    add_plus<2>(acc1, NXT.u1, NXT.a1, NXT.b1);
    // the y-neighbour inside the pair
    if (T.pair) add_plus<1>(acc0, CUR.u1, CUR.a1, CUR.b1);
    add_minus<1>(acc1, CUR.u0, CUR.a0, CUR.b0);
    __syncthreads();
    // (d) the other x / y neighbours from shared memory
    if (!T.pair) {                             // ragged tile: my second row is the halo row
      const float4 u = sU[buf][T.ly + 2][T.tx + 1]; const float2 ab = sAB[buf][T.ly + 2][T.tx + 1];
      add_plus<1>(acc0, u, ab.x, ab.y);
    }
    {
      const float4 u = sU[buf][T.ly + 1][T.tx]; const float2 ab = sAB[buf][T.ly + 1][T.tx];
      add_minus<0>(acc0, u, ab.x, ab.y);
    }
    {
      const float4 u = sU[buf][T.ly + 1][T.tx + 2]; const float2 ab = sAB[buf][T.ly + 1][T.tx + 2];
      add_plus<0>(acc0, u, ab.x, ab.y);
    }
    {
      const float4 u = sU[buf][T.ly][T.tx + 1]; const float2 ab = sAB[buf][T.ly][T.tx + 1];
      add_minus<1>(acc0, u, ab.x, ab.y);
    }
    {
      const float4 u = sU[buf][T.ly + 2][T.tx]; const float2 ab = sAB[buf][T.ly + 2][T.tx];
      add_minus<0>(acc1, u, ab.x, ab.y);
    }
    {
      const float4 u = sU[buf][T.ly + 2][T.tx + 2]; const float2 ab = sAB[buf][T.ly + 2][T.tx + 2];
      add_plus<0>(acc1, u, ab.x, ab.y);
    }
    {
      const float4 u = sU[buf][T.ly + 3][T.tx + 1]; const float2 ab = sAB[buf][T.ly + 3][T.tx + 1];
      add_plus<1>(acc1, u, ab.x, ab.y);
    }
    float4 o0, o1;
    mul2(o0.x, o0.y, CUR.u0.x, CUR.u0.y, c0, c0); mul2(o0.z, o0.w, CUR.u0.z, CUR.u0.w, c0, c0);
    mul2(o1.x, o1.y, CUR.u1.x, CUR.u1.y, c0, c0); mul2(o1.z, o1.w, CUR.u1.z, CUR.u1.w, c0, c0);
    fma2(o0.x, o0.y, acc0.x, acc0.y, c1, c1, o0.x, o0.y); fma2(o0.z, o0.w, acc0.z, acc0.w, c1, c1, o0.z, o0.w);
    fma2(o1.x, o1.y, acc1.x, acc1.y, c1, c1, o1.x, o1.y); fma2(o1.z, o1.w, acc1.z, acc1.w, c1, c1, o1.z, o1.w);
    if (T.act0) pst[0] = o0;
    if (T.act1) pst[d1] = o1;
    if (DIAG) {
      // non-finite scan and N dV total (chemistry off: no later kernel looks at the field)
      if (T.act0) {
        if (!(fabsf(o0.x) + fabsf(o0.y) + fabsf(o0.z) + fabsf(o0.w) < __int_as_float(0x7f800000))) acc_d.nonfinite++;
        acc_d.total += (double)o0.x;
      }
      if (T.act1) {
        if (!(fabsf(o1.x) + fabsf(o1.y) + fabsf(o1.z) + fabsf(o1.w) < __int_as_float(0x7f800000))) acc_d.nonfinite++;
        acc_d.total += (double)o1.x;
      }
    }
    if (OPEN) {
      // outflow through open faces (A15): transmissive face flux = own F_d (ghost copies the cell), reflective = 0
      if (T.act0) {
        if (x == 0 && p.bc[0] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)CUR.u0.y;
        if (x == n - 1 && p.bc[1] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)CUR.u0.y;
        if (y == 0 && p.bc[2] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)CUR.u0.z;
        if (y == n - 1 && p.bc[3] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)CUR.u0.z;
        if (z == 0 && p.bc[4] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)CUR.u0.w;
        if (z == n - 1 && p.bc[5] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)CUR.u0.w;
      }
      // inflow faces: the GLF face flux of Eq. 32 with the prescribed ghost, N-component (in units of c)
      auto in_lo = [&](const float4& c, float pc_, const float4& gst, float pg) { return 0.5 * ((double)pg + pc_) - 0.5 * ((double)c.x - gst.x); };
      auto in_hi = [&](const float4& c, float pc_, const float4& gst, float pg) { return 0.5 * ((double)pc_ + pg) - 0.5 * ((double)gst.x - c.x); };
      for (int k = 0; k < 2; k++) {
        const bool a = k ? T.act1 : T.act0;
        if (!a) continue;
        const float4& c = k ? CUR.u1 : CUR.u0;
        const int yy = y + k;
        if (x == 0 && p.bc[0] == EMMA_RT_BC_INFLOW) acc_d.outflow -= in_lo(c, c.y, p.inflow[0][g], p.inflow[0][g].y);
        if (x == n - 1 && p.bc[1] == EMMA_RT_BC_INFLOW) acc_d.outflow += in_hi(c, c.y, p.inflow[1][g], p.inflow[1][g].y);
        if (yy == 0 && p.bc[2] == EMMA_RT_BC_INFLOW) acc_d.outflow -= in_lo(c, c.z, p.inflow[2][g], p.inflow[2][g].z);
        if (yy == n - 1 && p.bc[3] == EMMA_RT_BC_INFLOW) acc_d.outflow += in_hi(c, c.z, p.inflow[3][g], p.inflow[3][g].z);
        if (z == 0 && p.bc[4] == EMMA_RT_BC_INFLOW) acc_d.outflow -= in_lo(c, c.w, p.inflow[4][g], p.inflow[4][g].w);
        if (z == n - 1 && p.bc[5] == EMMA_RT_BC_INFLOW) acc_d.outflow += in_hi(c, c.w, p.inflow[5][g], p.inflow[5][g].w);
      }
      if (T.act1) {
        if (x == 0 && p.bc[0] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)CUR.u1.y;
        if (x == n - 1 && p.bc[1] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)CUR.u1.y;
        if (y + 1 == n - 1 && p.bc[3] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)CUR.u1.z;
        if (z == 0 && p.bc[4] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)CUR.u1.w;
        if (z == n - 1 && p.bc[5] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)CUR.u1.w;
      }
    }
    // (e) this plane becomes the one below
    W0 = below_z(CUR.u0, CUR.a0, CUR.b0);
    W1 = below_z(CUR.u1, CUR.a1, CUR.b1);
    sg_nxt = last2 ? sgtop : 1.f;
    pld += plane; pst += plane;
    z++;
  };

  // the three register slots rotate roles, so the march is unrolled by three (no register moves, static buffers)
  for (;;) {
    body(A, B, C, 0); if (z >= z1) break;
    body(B, C, A, 1); if (z >= z1) break;
    body(C, A, B, 2); if (z >= z1) break;
  }

  if (DIAG || OPEN) {
    // photons: sums are in units of N; scale by nu dV (outflow = c phi dt dx^2 = nu phi dV) resp. dV
    acc_d.outflow *= (double)p.nu * p.dV;
    acc_d.total *= p.dV;
    block_reduce_store(acc_d, parts + blockIdx.x);
  }
}

}  // namespace

int launch_transport(const TransportParams& p, const float4* Uin, float4* Uout, Partial* parts, int* n_parts,
                     cudaStream_t st)
{
  const int nblk = p.tiles_x * p.tiles_y * p.nzc * p.G;
  bool open = false;
  for (int f = 0; f < 6; f++) open = open || (p.bc[f] == EMMA_RT_BC_TRANSMISSIVE) || (p.bc[f] == EMMA_RT_BC_INFLOW);
  const bool diag = p.want_total != 0;
  if (diag && open) transport_kernel<true, true><<<nblk, NT, 0, st>>>(p, Uin, Uout, parts);
  else if (diag) transport_kernel<true, false><<<nblk, NT, 0, st>>>(p, Uin, Uout, parts);
  else if (open) transport_kernel<false, true><<<nblk, NT, 0, st>>>(p, Uin, Uout, parts);
  else transport_kernel<false, false><<<nblk, NT, 0, st>>>(p, Uin, Uout, parts);
  *n_parts = (diag || open) ? nblk : 0;
  return 1;
}

}  // namespace emma
