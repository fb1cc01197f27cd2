// transport_hll.cu -- explicit M1 transport with the HLL interface flux.
//
// PAPER.md:250 names the HLL flux as the less diffusive successor of the GLF flux of Eq. 32 and prints nothing else;
// DESIGN.md reading A19 fixes it:  Eq. 30 with
//     H_{i+1/2} = [ l+ G_L - l- G_R + l+ l- (U_R - U_L) ] / (l+ - l-),   l+ = max(0, lmax_L, lmax_R),  l- = min(0, lmin_L, lmin_R),
// G_d = (phi_d, Pi_d.) the flux vector in the internal variables phi = F/c (units of N), l the extreme eigenvalues of
// dG_d/dU in units of c:
//     l(-/+) = [ r_d -/+ sqrt(R_d) ] / xi,   r = phi/N (scaled to |r| = 1 if f > 1),  xi = sqrt(4 - 3 f^2),
//     R_d = 2 (1 - f^2) (xi - 3 r_d^2 / (2 + xi)) / (xi + 1)
// -- algebraically the textbook radicand (2/3)(xi^2 - xi) + 2 mu^2 (2 - f^2 - xi) with mu f = r_d and
// (2 - xi)/f^2 = 3/(2 + xi); this form has no cancellation at f -> 1 and no 0/0 at f -> 0.  l+ = -l- = 1 gives Eq. 32.
// The update is U' = U - nu sum_d (H_{d+1/2} - H_{d-1/2}).  If l+ = l- (= 0: both cells stream exactly along the face)
// the flux vectors vanish too and H = 0.  The updated state is kept realizable (A19): |phi'| > N' -> phi' := max(N',0) phi'/|phi'|.
//
// Shape: one group per CTA; 256 threads own a column of 31 x 16 cells and march along z through a TMA-fed ring of planes
// (j-1, j, j+1 resident, the rest in flight), split-phase plane barrier as in fused.cu.  Every interface flux is evaluated
// ONCE where the layout allows it (3.5 faces per cell instead of 5):
//   * a thread owns the two cells (x, 2w) and (x, 2w+1): the y face between them is computed once, in registers; the y faces
//     towards the rows of the neighbouring warps are computed by both sides (no exchange, no extra barrier);
//   * the 32 lanes of a warp hold the tile's LEFT HALO cell (lane 0) and its 31 cells (lanes 1..31); every lane computes
//     the face on its right, and the face on a cell's left arrives from the lane below by shuffle.  Lane 0 updates nothing:
//     tiles are 31 cells wide so that no warp runs a whole face evaluation for one boundary lane;
//   * the z face is carried from plane to plane.
// Per cell the closure (a, b) and the six wave speeds are computed ONCE, when its plane lands, and staged in shared
// memory beside U (32 B per cell).
#include <cuda.h>

#include "async_copy.cuh"
#include "emma_rt_internal.cuh"
#include "transport_math.cuh"
#include "hll_math.cuh"

namespace emma {

namespace {

using namespace acp;

constexpr int TXC = 31;                        // cells per tile row that this CTA updates (lanes 1..31)
constexpr int TY = 16, NW = TY / 2, NT = 32 * NW;
constexpr int TXM = TXC + 2;                   // the main box also brings the x halo: cells x0-1 .. x0+31, cell x0+l-1 in slot l
constexpr int ROWB = TXM * 16;                 // bytes of one row of the main box (dense: what the TMA delivers)
constexpr int COLB = TY * 16;                  // bytes of one halo column
// One plane: [MAIN 16 x 33][BOT 31][TOP 31][LCOL 16][RCOL 16] cells, every box at a 128-byte aligned offset (TMA).  With the
// x halo inside the rows a quarter-warp reads 128 contiguous bytes (any 16-byte phase): no bank conflict; a halo taken from
// a separate column box costs one more wavefront per load (profiles/r2e_hll_summary.md: 29 % of the shared-memory
// wavefronts).  LCOL / RCOL are read only by the tiles on a box face, where the halo is a periodic image or a ghost.
constexpr int MAIN = 0, BOT = TY * ROWB, TOP = BOT + 512, LCOL = TOP + 512, RCOL = LCOL + COLB;
constexpr int SG = RCOL + COLB;                // bytes of one plane (9984 = 78 x 128)
static_assert(BOT % 128 == 0 && SG % 128 == 0, "TMA destinations must be 128-byte aligned");
constexpr int NST = 6;                         // stages of the ring
constexpr int AUXB = 2 * SG;                   // aux plane: two sub-planes of one float4 per cell, each laid out like a stage
constexpr size_t SMEM = (size_t)NST * SG + 2 * AUXB + 8 * (NST + 1);

__device__ __forceinline__ void store_aux(unsigned char* plane, int off, const Aux& A)
{
  *(float4*)(plane + off) = make_float4(A.a, A.b, A.lm[0], A.lp[0]);
  *(float4*)(plane + SG + off) = make_float4(A.lm[1], A.lp[1], A.lm[2], A.lp[2]);
}
__device__ __forceinline__ float4 shfl_up4(const float4& v)
{
  return make_float4(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1),
                     __shfl_up_sync(0xffffffffu, v.z, 1), __shfl_up_sync(0xffffffffu, v.w, 1));
}

// DIAG: chemistry is off, so this pass owns the step's photon total and non-finite scan.
// BCGEN: some face is not periodic (outflow sums and the reflective signs are compiled in).
template <bool DIAG, bool BCGEN>
__global__ void __launch_bounds__(NT, 2)
transport_hll_kernel(const TransportParams p, const __grid_constant__ TransportMaps maps, float4* __restrict__ Uout,
                     Partial* __restrict__ parts)
{
  extern __shared__ __align__(128) unsigned char smem[];
  unsigned char* const sAUX = smem + NST * SG;
  const unsigned bar0 = smem_u32(sAUX + 2 * AUXB);
  const unsigned bar_pl = bar0 + 8 * NST;      // split-phase "plane done" barrier (see fused.cu)
  const unsigned stage0 = smem_u32(smem);

  const int n = p.n;
  int bid = blockIdx.x;
  const int tix = bid % p.tiles_x; bid /= p.tiles_x;
  const int tiy = bid % p.tiles_y; bid /= p.tiles_y;
  const int izc = bid % p.nzc;     bid /= p.nzc;
  const int g = bid;
  const int x0 = tix * TXC, y0 = tiy * TY;
  const int wx = min(TXC, n - x0), wy = min(TY, n - y0);
  const int z0 = izc * p.zchunk, z1 = min(n, z0 + p.zchunk);
  const int zc = z1 - z0;
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const int r0 = 2 * warp;                     // my rows: r0 and r0 + 1
  const int x = x0 + lane - 1, y = y0 + r0;    // lane 0 holds the cell LEFT of the tile (never updated)
  const bool pair = r0 + 1 < wy;               // warp-uniform
  const bool col = lane >= 1 && lane <= wx;
  const bool act0 = col && r0 < wy, act1 = col && pair;
  const bool ghostL = BCGEN && lane == 0 && x0 == 0 && p.bc[0] != EMMA_RT_BC_PERIODIC;   // my cells are ghosts of the -x face

  // byte offsets inside a plane.  edgeL / edgeR: the tile touches the -x / +x face of the box, its halo there is not the
  // neighbour in memory (periodic image, ghost; also the ragged last tile): it comes from the column boxes
  const bool edgeL = x0 == 0, edgeR = x0 + wx == n;
  const int c16 = lane * 16;
  const int own0 = (lane == 0 && edgeL) ? LCOL + r0 * 16 : MAIN + r0 * ROWB + c16;
  const int own1 = (lane == 0 && edgeL) ? LCOL + (r0 + 1) * 16 : MAIN + (r0 + 1) * ROWB + c16;
  const int oxp0 = (lane >= wx && edgeR) ? RCOL + r0 * 16 : MAIN + r0 * ROWB + c16 + 16;
  const int oxp1 = (lane >= wx && edgeR) ? RCOL + (r0 + 1) * 16 : MAIN + (r0 + 1) * ROWB + c16 + 16;
  const int cl = (lane == 0) ? 1 : lane;       // lane 0 needs no y faces: any valid column
  const int oym0 = (r0 == 0) ? BOT + (cl - 1) * 16 : MAIN + (r0 - 1) * ROWB + cl * 16;
  const int oyp = (r0 + (pair ? 2 : 1) < wy) ? MAIN + (r0 + 2) * ROWB + cl * 16 : TOP + (cl - 1) * 16;   // above my upper cell
  float sxp = 1.f, sym = 1.f, syp = 1.f;       // reflective faces: sign of the face-normal flux of that neighbour (A13)
  if (BCGEN) {
    if (lane == wx && x0 + wx == n && p.bc[1] == EMMA_RT_BC_REFLECTIVE) sxp = -1.f;
    if (r0 == 0 && y0 == 0 && p.bc[2] == EMMA_RT_BC_REFLECTIVE) sym = -1.f;
    if (r0 + (pair ? 2 : 1) == wy && y0 + wy == n && p.bc[3] == EMMA_RT_BC_REFLECTIVE) syp = -1.f;
  }
  // the ghost of the -x face that lane 0 holds: the cell itself mirrored (reflective), as it is (transmissive), or the
  // prescribed inflow state (A13, A20)
  auto ghost_left = [&](float4& u) {
    if (ghostL) {
      if (p.bc[0] == EMMA_RT_BC_INFLOW) u = p.inflow[0][g];
      else if (p.bc[0] == EMMA_RT_BC_REFLECTIVE) u.y = -u.y;
    }
  };
  // halo cells other than the left column: right column, bottom row, top row, dealt in order (task h -> thread h: whole
  // warps); a reflective ghost gets its aux from the mirrored state, an inflow ghost is the prescribed state
  int hoff = -1;
  float hsx = 1.f, hsy = 1.f;
  bool hin = false;
  float4 hval = make_float4(0.f, 0.f, 0.f, 0.f);
  {
    const int nh = wy + 2 * wx, h = t;
    if (h < nh) {
      int face;
      if (h < wy) { hoff = edgeR ? RCOL + h * 16 : MAIN + h * ROWB + (TXC + 1) * 16; face = edgeR ? 1 : -1; }
      else if (h < wy + wx) { hoff = BOT + (h - wy) * 16; face = (y0 == 0) ? 2 : -1; }
      else { hoff = TOP + (h - wy - wx) * 16; face = (y0 + wy == n) ? 3 : -1; }
      if (BCGEN && face >= 0) {
        if (p.bc[face] == EMMA_RT_BC_INFLOW) { hin = true; hval = p.inflow[face][g]; }
        else if (p.bc[face] == EMMA_RT_BC_REFLECTIVE) { if (face == 1) hsx = -1.f; else hsy = -1.f; }
      }
    }
  }

  const bool zin_lo = BCGEN && z0 == 0 && p.bc[4] == EMMA_RT_BC_INFLOW;
  const bool zin_hi = BCGEN && z1 == n && p.bc[5] == EMMA_RT_BC_INFLOW;
  bool flz, fltop, fl;
  const int zm = bc_map(z0 - 1, n, p.bc[4], p.bc[5], flz);
  const int ztop = bc_map(z1, n, p.bc[4], p.bc[5], fltop);
  const int cxl = 4 * bc_map(x0 - 1, n, p.bc[0], p.bc[1], fl);
  const int cxr = 4 * bc_map(x0 + wx, n, p.bc[0], p.bc[1], fl);
  const int cyb = bc_map(y0 - 1, n, p.bc[2], p.bc[3], fl);
  const int cyt = bc_map(y0 + wy, n, p.bc[2], p.bc[3], fl);

  auto issue = [&](int j, int s) {             // the five boxes of plane j, each by the first lane of a different warp
    if (lane != 0 || warp >= 5) return;
    const int zg = g * n + ((j < 0) ? zm : (j >= zc) ? ztop : z0 + j);
    const unsigned bar = bar0 + 8 * s, dst = stage0 + s * SG;
    if (warp == 0) { mbar_expect_tx(bar, TY * ROWB); tma_load_3d(dst + MAIN, &maps.main, bar, 4 * (x0 - 1), y0, zg); }
    else if (warp == 1) { mbar_expect_tx(bar, TXC * 16); tma_load_3d(dst + BOT, &maps.row, bar, 4 * x0, cyb, zg); }
    else if (warp == 2) { mbar_expect_tx(bar, TXC * 16); tma_load_3d(dst + TOP, &maps.row, bar, 4 * x0, cyt, zg); }
    else if (warp == 3) { mbar_expect_tx(bar, COLB); tma_load_3d(dst + LCOL, &maps.col, bar, cxl, y0, zg); }
    else { mbar_expect_tx(bar, COLB); tma_load_3d(dst + RCOL, &maps.col, bar, cxr, y0, zg); }
  };

  if (t == 0) {
    for (int s = 0; s < NST; s++) mbar_init(bar0 + 8 * s, 5);
    mbar_init(bar_pl, NT / 32);
    mbar_fence_init();
  }
  __syncthreads();
  for (int j = -1; j < NST - 1 && j <= zc; j++) issue(j, j + 1);

  const float nu = p.nu;
  const size_t plane = (size_t)n * n;
  float4* pst = Uout + ((size_t)g * n + z0) * plane + (act0 ? ((size_t)y * n + x) : 0);
  const ptrdiff_t d1 = act1 ? n : 0;
  Acc acc_d;

  auto halo_aux = [&](unsigned char* st, unsigned char* aux) {
    if (hoff >= 0) {
      float4 h = *(const float4*)(st + hoff);
      if (BCGEN && hin) { h = hval; *(float4*)(st + hoff) = h; }        // consumers read the ghost from the stage
      if (BCGEN) { h.y *= hsx; h.z *= hsy; }
      store_aux(aux, hoff, make_aux(h));
    }
  };
  // my two cells of the plane in stage `st` (lane 0: the ghosts / periodic images left of the tile)
  auto load_own = [&](const unsigned char* st, float4& u0, float4& u1) {
    u0 = *(const float4*)(st + own0); u1 = *(const float4*)(st + own1);
    if (BCGEN) { ghost_left(u0); ghost_left(u1); }
  };

  // ---- prologue: aux of plane -1 (own cells only: it is only ever a z-neighbour) and of plane 0
  {
    mbar_wait(bar0, 0);
    float4 m0, m1;
    load_own(smem, m0, m1);
    if (BCGEN && zin_lo) { m0 = p.inflow[4][g]; m1 = m0; }
    if (BCGEN && flz) { m0.w = -m0.w; m1.w = -m1.w; }
    store_aux(sAUX, own0, make_aux(m0)); store_aux(sAUX, own1, make_aux(m1));
    mbar_wait(bar0 + 8, 0);
    load_own(smem + SG, m0, m1);
    store_aux(sAUX + AUXB, own0, make_aux(m0)); store_aux(sAUX + AUXB, own1, make_aux(m1));
    halo_aux(smem + SG, sAUX + AUXB);
  }
  __syncthreads();

  int s_old = 0, s_blw = 0, s_cur = 1, s_nxt = 2 % NST;
  unsigned par_nxt = (2 / NST) & 1;
  int ab_blw = 0, ab_cur = 1;
  float4 Hzm0 = make_float4(0.f, 0.f, 0.f, 0.f), Hzm1 = Hzm0;

  for (int j = 0; j < zc; j++) {
    if (j > 0) {
      mbar_wait_relaxed(bar_pl, (unsigned)(j - 1) & 1u);
      if (j + NST - 2 <= zc) issue(j + NST - 2, s_old);
    }
    const unsigned char* sb = smem + s_blw * SG;
    const unsigned char* sc = smem + s_cur * SG;
    unsigned char* sn = smem + s_nxt * SG;
    unsigned char* AXb = sAUX + ab_blw * AUXB;                         // aux of plane j-1; receives plane j+1
    const unsigned char* AXc = sAUX + ab_cur * AUXB;
    mbar_wait(bar0 + 8 * s_nxt, par_nxt);
    const bool top = (j + 1 == zc);

    // my cells and their aux (staged by me one plane ago): [a, b, lmx, lpx], [lmy, lpy, lmz, lpz]
    float4 cu0, cu1, un0, un1;
    load_own(sc, cu0, cu1);
    const float4 a0 = *(const float4*)(AXc + own0), b0 = *(const float4*)(AXc + SG + own0);
    const float4 a1 = *(const float4*)(AXc + own1), b1 = *(const float4*)(AXc + SG + own1);
    // the plane above: aux now (kept for the z face, staged for the next plane)
    load_own(sn, un0, un1);
    if (BCGEN && top && zin_hi) { un0 = p.inflow[5][g]; un1 = un0; }
    if (BCGEN && top && fltop) { un0.w = -un0.w; un1.w = -un1.w; }
    const Aux An0 = make_aux(un0), An1 = make_aux(un1);
    if (j == 0) {
      // the face below the chunk: flux from the plane below (afterwards it is carried from plane to plane)
      float4 ub0, ub1;
      load_own(sb, ub0, ub1);
      if (BCGEN && zin_lo) { ub0 = p.inflow[4][g]; ub1 = ub0; }
      if (BCGEN && flz) { ub0.w = -ub0.w; ub1.w = -ub1.w; }
      const float4 q0 = *(const float4*)(AXb + own0), r0v = *(const float4*)(AXb + SG + own0);
      const float4 q1 = *(const float4*)(AXb + own1), r1v = *(const float4*)(AXb + SG + own1);
      Hzm0 = hll_face<2>(ub0, q0.x, q0.y, r0v.z, r0v.w, cu0, a0.x, a0.y, b0.z, b0.w);
      Hzm1 = hll_face<2>(ub1, q1.x, q1.y, r1v.z, r1v.w, cu1, a1.x, a1.y, b1.z, b1.w);
    }
    if (!top) {
      store_aux(AXb, own0, An0); store_aux(AXb, own1, An1);
      halo_aux(sn, AXb);
    }
    const float4 Hzp0 = hll_face<2>(cu0, a0.x, a0.y, b0.z, b0.w, un0, An0.a, An0.b, An0.lm[2], An0.lp[2]);
    const float4 Hzp1 = hll_face<2>(cu1, a1.x, a1.y, b1.z, b1.w, un1, An1.a, An1.b, An1.lm[2], An1.lp[2]);
    // x: every lane evaluates the face on its RIGHT; the face on a cell's left comes from the lane below
    float4 u, q;
    float2 r;
    u = *(const float4*)(sc + oxp0); q = *(const float4*)(AXc + oxp0); if (BCGEN) u.y *= sxp;
    const float4 Hxp0 = hll_face<0>(cu0, a0.x, a0.y, a0.z, a0.w, u, q.x, q.y, q.z, q.w);
    u = *(const float4*)(sc + oxp1); q = *(const float4*)(AXc + oxp1); if (BCGEN) u.y *= sxp;
    const float4 Hxp1 = hll_face<0>(cu1, a1.x, a1.y, a1.z, a1.w, u, q.x, q.y, q.z, q.w);
    const float4 Hxm0 = shfl_up4(Hxp0), Hxm1 = shfl_up4(Hxp1);
    // y: below my lower cell, between my two cells (once), above my upper cell
    u = *(const float4*)(sc + oym0); q = *(const float4*)(AXc + oym0); r = *(const float2*)(AXc + SG + oym0); if (BCGEN) u.z *= sym;
    const float4 Hym0 = hll_face<1>(u, q.x, q.y, r.x, r.y, cu0, a0.x, a0.y, b0.x, b0.y);
    u = *(const float4*)(sc + oyp); q = *(const float4*)(AXc + oyp); r = *(const float2*)(AXc + SG + oyp); if (BCGEN) u.z *= syp;
    float4 Hyp0, Hyp1 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (pair) {
      Hyp0 = hll_face<1>(cu0, a0.x, a0.y, b0.x, b0.y, cu1, a1.x, a1.y, b1.x, b1.y);
      Hyp1 = hll_face<1>(cu1, a1.x, a1.y, b1.x, b1.y, u, q.x, q.y, r.x, r.y);
    } else {
      Hyp0 = hll_face<1>(cu0, a0.x, a0.y, b0.x, b0.y, u, q.x, q.y, r.x, r.y);
    }
    // my reads of planes j-1, j and my aux writes of plane j+1 are done
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_pl);

    auto update = [&](const float4& cu, const float4& Hxm, const float4& Hxp, const float4& Hym, const float4& Hyp,
                      const float4& Hzm, const float4& Hzp) -> float4 {
      // Eq. 30, unsplit (A4): o = cu - nu [(Hxp - Hxm) + (Hyp - Hym) + (Hzp - Hzm)], on the (N, phi_x) and (phi_y, phi_z) halves
      float4 o, dx, dy, dz;
      sub2(dx.x, dx.y, Hxp.x, Hxp.y, Hxm.x, Hxm.y); sub2(dx.z, dx.w, Hxp.z, Hxp.w, Hxm.z, Hxm.w);
      sub2(dy.x, dy.y, Hyp.x, Hyp.y, Hym.x, Hym.y); sub2(dy.z, dy.w, Hyp.z, Hyp.w, Hym.z, Hym.w);
      sub2(dz.x, dz.y, Hzp.x, Hzp.y, Hzm.x, Hzm.y); sub2(dz.z, dz.w, Hzp.z, Hzp.w, Hzm.z, Hzm.w);
      fma2(dx.x, dx.y, dx.x, dx.y, 1.f, 1.f, dy.x, dy.y); fma2(dx.z, dx.w, dx.z, dx.w, 1.f, 1.f, dy.z, dy.w);
      fma2(dx.x, dx.y, dx.x, dx.y, 1.f, 1.f, dz.x, dz.y); fma2(dx.z, dx.w, dx.z, dx.w, 1.f, 1.f, dz.z, dz.w);
      fma2(o.x, o.y, dx.x, dx.y, -nu, -nu, cu.x, cu.y); fma2(o.z, o.w, dx.z, dx.w, -nu, -nu, cu.z, cu.w);
      // A19: keep the state realizable, |phi| <= max(N, 0)
      const float p2 = fmaf(o.y, o.y, fmaf(o.z, o.z, o.w * o.w)), Np = fmaxf(o.x, 0.f);
      if (p2 > Np * Np) { const float sc = Np * rsqrtf(p2); o.y *= sc; o.z *= sc; o.w *= sc; }
      return o;
    };
    const float4 o0 = update(cu0, Hxm0, Hxp0, Hym0, Hyp0, Hzm0, Hzp0);
    const float4 o1 = update(cu1, Hxm1, Hxp1, Hyp0, Hyp1, Hzm1, Hzp1);
    if (act0) pst[0] = o0;
    if (act1) pst[d1] = o1;
    if (DIAG) {
      if (act0) {
        if (!(fabsf(o0.x) + fabsf(o0.y) + fabsf(o0.z) + fabsf(o0.w) < __int_as_float(0x7f800000))) acc_d.nonfinite++;
        acc_d.total += (double)o0.x;
      }
      if (act1) {
        if (!(fabsf(o1.x) + fabsf(o1.y) + fabsf(o1.z) + fabsf(o1.w) < __int_as_float(0x7f800000))) acc_d.nonfinite++;
        acc_d.total += (double)o1.x;
      }
    }
    if (BCGEN) {
      // outflow through non-periodic faces (A15): the N-component of the face fluxes just evaluated (transmissive:
      // the cell's own phi_d; reflective: 0 up to rounding; inflow: negative while light enters)
      const int z = z0 + j;
      if (act0) {
        if (x == 0 && p.bc[0] != EMMA_RT_BC_PERIODIC) acc_d.outflow -= (double)Hxm0.x;
        if (x == n - 1 && p.bc[1] != EMMA_RT_BC_PERIODIC) acc_d.outflow += (double)Hxp0.x;
        if (y == 0 && p.bc[2] != EMMA_RT_BC_PERIODIC) acc_d.outflow -= (double)Hym0.x;
        if (y == n - 1 && p.bc[3] != EMMA_RT_BC_PERIODIC) acc_d.outflow += (double)Hyp0.x;
        if (z == 0 && p.bc[4] != EMMA_RT_BC_PERIODIC) acc_d.outflow -= (double)Hzm0.x;
        if (z == n - 1 && p.bc[5] != EMMA_RT_BC_PERIODIC) acc_d.outflow += (double)Hzp0.x;
      }
      if (act1) {
        if (x == 0 && p.bc[0] != EMMA_RT_BC_PERIODIC) acc_d.outflow -= (double)Hxm1.x;
        if (x == n - 1 && p.bc[1] != EMMA_RT_BC_PERIODIC) acc_d.outflow += (double)Hxp1.x;
        if (y + 1 == n - 1 && p.bc[3] != EMMA_RT_BC_PERIODIC) acc_d.outflow += (double)Hyp1.x;
        if (z == 0 && p.bc[4] != EMMA_RT_BC_PERIODIC) acc_d.outflow -= (double)Hzm1.x;
        if (z == n - 1 && p.bc[5] != EMMA_RT_BC_PERIODIC) acc_d.outflow += (double)Hzp1.x;
      }
    }
    Hzm0 = Hzp0; Hzm1 = Hzp1;
    pst += plane;
    s_old = s_blw; s_blw = s_cur; s_cur = s_nxt;
    if (++s_nxt == NST) { s_nxt = 0; par_nxt ^= 1u; }
    const int ab_nxt = ab_blw;
    ab_blw = ab_cur; ab_cur = ab_nxt;
  }

  if (DIAG || BCGEN) {
    acc_d.outflow *= (double)p.nu * p.dV;
    acc_d.total *= p.dV;
    block_reduce_store(acc_d, parts + blockIdx.x);
  }
}

template <bool DIAG, bool BCGEN>
cudaError_t launch_variant(const TransportParams& p, const TransportMaps& maps, float4* Uout, Partial* parts, int nblk,
                           cudaStream_t st)
{
  transport_hll_kernel<DIAG, BCGEN><<<nblk, NT, SMEM, st>>>(p, maps, Uout, parts);
  return cudaSuccess;
}

}  // namespace

// Per-device set-up (emma_rt_init, handle's device current): dynamic shared memory opt-in
cudaError_t configure_transport_hll()
{
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(transport_hll_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(transport_hll_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(transport_hll_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM)) != cudaSuccess) return e;
  return cudaFuncSetAttribute(transport_hll_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM);
}

int hll_ctas_per_sm() { return 2; }
int hll_tile_x() { return TXC; }
int hll_main_x() { return TXM; }

int launch_transport_hll(const TransportParams& p, const TransportMaps& maps_in, float4* Uout, Partial* parts,
                         int* n_parts, cudaStream_t st)
{
  const int nblk = p.tiles_x * p.tiles_y * p.nzc * p.G;
  bool bcgen = false;
  for (int f = 0; f < 6; f++) bcgen = bcgen || (p.bc[f] != EMMA_RT_BC_PERIODIC);
  const bool diag = p.want_total != 0;
  cudaError_t e;
  if (diag && bcgen) e = launch_variant<true, true>(p, maps_in, Uout, parts, nblk, st);
  else if (diag) e = launch_variant<true, false>(p, maps_in, Uout, parts, nblk, st);
  else if (bcgen) e = launch_variant<false, true>(p, maps_in, Uout, parts, nblk, st);
  else e = launch_variant<false, false>(p, maps_in, Uout, parts, nblk, st);
  *n_parts = (diag || bcgen) ? nblk : 0;
  return e == cudaSuccess ? 1 : 0;
}

}  // namespace emma
