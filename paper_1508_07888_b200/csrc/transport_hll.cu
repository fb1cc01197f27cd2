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
// Shape: as fused.cu with one group per CTA -- 512 threads own a 32 x 16 column, one cell each, and march along z
// through a TMA-fed ring of planes (j-1, j, j+1 resident, the rest in flight).  Per cell the closure (a, b) and the six
// wave speeds are computed ONCE, when its plane lands, and staged in shared memory (32 B per cell); the x/y face
// fluxes are evaluated from both sides (once per adjacent cell), the z face flux is carried to the next plane.
#include <cuda.h>

#include "async_copy.cuh"
#include "emma_rt_internal.cuh"
#include "transport_math.cuh"
#include "hll_math.cuh"

namespace emma {

namespace {

using namespace acp;

constexpr int TX = 32, TY = 16, NT = TX * TY;
constexpr int ROWB = TX * 16;
constexpr int TOPROW = (TY + 1) * ROWB;
constexpr int STAGE_ROWS = (TY + 2) * ROWB;
constexpr int COLB = TY * 16;
constexpr int SG = STAGE_ROWS + 2 * COLB;      // bytes of one plane (own 32 x 16 box, 2 halo rows, 2 halo columns)
constexpr int NST = 6;                         // stages of the ring
constexpr int AUXB = 2 * SG;                   // aux plane: two sub-planes of one float4 per cell, each laid out like a stage
                                               // (consecutive lanes -> consecutive 16 B: no bank conflicts)
constexpr size_t SMEM = (size_t)NST * SG + 2 * AUXB + 8 * (NST + 1);

__device__ __forceinline__ void store_aux(unsigned char* plane, int off, const Aux& A)
{
  *(float4*)(plane + off) = make_float4(A.a, A.b, A.lm[0], A.lp[0]);
  *(float4*)(plane + SG + off) = make_float4(A.lm[1], A.lp[1], A.lm[2], A.lp[2]);
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
  const int x0 = tix * TX, y0 = tiy * TY;
  const int wx = min(TX, n - x0), wy = min(TY, n - y0);
  const int z0 = izc * p.zchunk, z1 = min(n, z0 + p.zchunk);
  const int zc = z1 - z0;
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const int tx = t % TX, ty = t / TX;
  const int x = x0 + tx, y = y0 + ty;
  const bool act = (tx < wx) && (ty < wy);

  const int own = (ty + 1) * ROWB + tx * 16;
  const int oxm = (tx > 0) ? own - 16 : STAGE_ROWS + ty * 16;
  const int oxp = (tx < wx - 1) ? own + 16 : STAGE_ROWS + COLB + ty * 16;
  const int oym = own - ROWB;
  const int oyp = (ty + 1 < wy) ? own + ROWB : TOPROW + tx * 16;
  float sxm = 1.f, sxp = 1.f, sym = 1.f, syp = 1.f;     // reflective faces: sign of the face-normal flux (A13)
  if (BCGEN) {
    if (tx == 0 && x0 == 0 && p.bc[0] == EMMA_RT_BC_REFLECTIVE) sxm = -1.f;
    if (tx == wx - 1 && x0 + wx == n && p.bc[1] == EMMA_RT_BC_REFLECTIVE) sxp = -1.f;
    if (ty == 0 && y0 == 0 && p.bc[2] == EMMA_RT_BC_REFLECTIVE) sym = -1.f;
    if (ty == wy - 1 && y0 + wy == n && p.bc[3] == EMMA_RT_BC_REFLECTIVE) syp = -1.f;
  }
  // halo cells: dealt in order, task h -> thread h (96 tasks = 3 whole warps; the others skip the work, and consecutive
  // lanes read consecutive cells); a reflective ghost gets its aux from the mirrored state (face-normal component negated)
  int hoff = -1;
  float hsx = 1.f, hsy = 1.f;
  bool hin = false;                            // my halo cell is the ghost of an inflow face (A20): a prescribed state
  float4 hval = make_float4(0.f, 0.f, 0.f, 0.f);
  {
    const int nh = 2 * wy + 2 * wx, h = t;
    if (BCGEN && h < nh) {
      const int face = (h < wy) ? (x0 == 0 ? 0 : -1) : (h < 2 * wy) ? (x0 + wx == n ? 1 : -1)
                     : (h < 2 * wy + wx) ? (y0 == 0 ? 2 : -1) : (y0 + wy == n ? 3 : -1);
      if (face >= 0 && p.bc[face] == EMMA_RT_BC_INFLOW) { hin = true; hval = p.inflow[face][g]; }
    }
    if (h < nh) {
      if (h < wy) { hoff = STAGE_ROWS + h * 16; if (BCGEN && x0 == 0 && p.bc[0] == EMMA_RT_BC_REFLECTIVE) hsx = -1.f; }
      else if (h < 2 * wy) { hoff = STAGE_ROWS + COLB + (h - wy) * 16; if (BCGEN && x0 + wx == n && p.bc[1] == EMMA_RT_BC_REFLECTIVE) hsx = -1.f; }
      else if (h < 2 * wy + wx) { hoff = (h - 2 * wy) * 16; if (BCGEN && y0 == 0 && p.bc[2] == EMMA_RT_BC_REFLECTIVE) hsy = -1.f; }
      else { hoff = TOPROW + (h - 2 * wy - wx) * 16; if (BCGEN && y0 + wy == n && p.bc[3] == EMMA_RT_BC_REFLECTIVE) hsy = -1.f; }
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
    if (warp == 0) { mbar_expect_tx(bar, TY * ROWB); tma_load_3d(dst + ROWB, &maps.main, bar, 4 * x0, y0, zg); }
    else if (warp == 1) { mbar_expect_tx(bar, ROWB); tma_load_3d(dst, &maps.row, bar, 4 * x0, cyb, zg); }
    else if (warp == 2) { mbar_expect_tx(bar, ROWB); tma_load_3d(dst + TOPROW, &maps.row, bar, 4 * x0, cyt, zg); }
    else if (warp == 3) { mbar_expect_tx(bar, COLB); tma_load_3d(dst + STAGE_ROWS, &maps.col, bar, cxl, y0, zg); }
    else { mbar_expect_tx(bar, COLB); tma_load_3d(dst + STAGE_ROWS + COLB, &maps.col, bar, cxr, y0, zg); }
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
  float4* pst = Uout + ((size_t)g * n + z0) * plane + (act ? ((size_t)y * n + x) : 0);
  Acc acc_d;

  auto halo_aux = [&](unsigned char* st, unsigned char* aux) {
    if (hoff >= 0) {
      float4 h = *(const float4*)(st + hoff);
      if (BCGEN && hin) { h = hval; *(float4*)(st + hoff) = h; }        // consumers read the ghost from the stage
      if (BCGEN) { h.y *= hsx; h.z *= hsy; }
      store_aux(aux, hoff, make_aux(h));
    }
  };

  // ---- prologue: aux of plane -1 (own cells only: it is only ever a z-neighbour) and of plane 0
  {
    mbar_wait(bar0, 0);
    float4 m = *(const float4*)(smem + own);
    if (BCGEN && zin_lo) m = p.inflow[4][g];
    if (BCGEN && flz) m.w = -m.w;
    store_aux(sAUX, own, make_aux(m));
    mbar_wait(bar0 + 8, 0);
    store_aux(sAUX + AUXB, own, make_aux(*(const float4*)(smem + SG + own)));
    halo_aux(smem + SG, sAUX + AUXB);
  }
  __syncthreads();

  int s_old = 0, s_blw = 0, s_cur = 1, s_nxt = 2 % NST;
  unsigned par_nxt = (2 / NST) & 1;
  int ab_blw = 0, ab_cur = 1;
  float4 Hzm = make_float4(0.f, 0.f, 0.f, 0.f);

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

    // my cell and its aux (staged by me one plane ago)
    const float4 cu = *(const float4*)(sc + own);
    const float4 c0 = *(const float4*)(AXc + own), c1 = *(const float4*)(AXc + SG + own);
    // the plane above: aux now (kept for the z face, staged for the next plane)
    float4 un = *(const float4*)(sn + own);
    if (BCGEN && top && zin_hi) un = p.inflow[5][g];
    if (BCGEN && top && fltop) un.w = -un.w;
    const Aux An = make_aux(un);
    if (j == 0) {
      // the face below the chunk: flux from the plane below (afterwards it is carried from plane to plane)
      float4 ub = *(const float4*)(sb + own);
      if (BCGEN && zin_lo) ub = p.inflow[4][g];
      if (BCGEN && flz) ub.w = -ub.w;
      const float4 b0 = *(const float4*)(AXb + own), b1 = *(const float4*)(AXb + SG + own);
      Hzm = hll_face<2>(ub, b0.x, b0.y, b1.z, b1.w, cu, c0.x, c0.y, c1.z, c1.w);
    }
    if (!top) {
      store_aux(AXb, own, An);
      halo_aux(sn, AXb);
    }
    const float4 Hzp = hll_face<2>(cu, c0.x, c0.y, c1.z, c1.w, un, An.a, An.b, An.lm[2], An.lp[2]);
    float4 u, q;
    float2 r;
    u = *(const float4*)(sc + oxm); q = *(const float4*)(AXc + oxm); if (BCGEN) u.y *= sxm;
    const float4 Hxm = hll_face<0>(u, q.x, q.y, q.z, q.w, cu, c0.x, c0.y, c0.z, c0.w);
    u = *(const float4*)(sc + oxp); q = *(const float4*)(AXc + oxp); if (BCGEN) u.y *= sxp;
    const float4 Hxp = hll_face<0>(cu, c0.x, c0.y, c0.z, c0.w, u, q.x, q.y, q.z, q.w);
    u = *(const float4*)(sc + oym); q = *(const float4*)(AXc + oym); r = *(const float2*)(AXc + SG + oym); if (BCGEN) u.z *= sym;
    const float4 Hym = hll_face<1>(u, q.x, q.y, r.x, r.y, cu, c0.x, c0.y, c1.x, c1.y);
    u = *(const float4*)(sc + oyp); q = *(const float4*)(AXc + oyp); r = *(const float2*)(AXc + SG + oyp); if (BCGEN) u.z *= syp;
    const float4 Hyp = hll_face<1>(cu, c0.x, c0.y, c1.x, c1.y, u, q.x, q.y, r.x, r.y);
    // my reads of planes j-1, j and my aux writes of plane j+1 are done
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_pl);

    float4 o;                                                          // Eq. 30, unsplit (A4)
    o.x = fmaf(-nu, (Hxp.x - Hxm.x) + (Hyp.x - Hym.x) + (Hzp.x - Hzm.x), cu.x);
    o.y = fmaf(-nu, (Hxp.y - Hxm.y) + (Hyp.y - Hym.y) + (Hzp.y - Hzm.y), cu.y);
    o.z = fmaf(-nu, (Hxp.z - Hxm.z) + (Hyp.z - Hym.z) + (Hzp.z - Hzm.z), cu.z);
    o.w = fmaf(-nu, (Hxp.w - Hxm.w) + (Hyp.w - Hym.w) + (Hzp.w - Hzm.w), cu.w);
    const float Hz_lo = Hzm.x;
    {                                          // A19: keep the state realizable, |phi| <= max(N, 0)
      const float p2 = fmaf(o.y, o.y, fmaf(o.z, o.z, o.w * o.w)), Np = fmaxf(o.x, 0.f);
      if (p2 > Np * Np) { const float sc = Np * rsqrtf(p2); o.y *= sc; o.z *= sc; o.w *= sc; }
    }
    Hzm = Hzp;
    if (act) {
      *pst = o;
      if (DIAG) {
        if (!(fabsf(o.x) + fabsf(o.y) + fabsf(o.z) + fabsf(o.w) < __int_as_float(0x7f800000))) acc_d.nonfinite++;
        acc_d.total += (double)o.x;
      }
      if (BCGEN) {
        // outflow through non-periodic faces (A15): the N-component of the face fluxes just evaluated (transmissive:
        // the cell's own phi_d; reflective: 0 up to rounding; inflow: negative while light enters)
        const int z = z0 + j;
        if (x == 0 && p.bc[0] != EMMA_RT_BC_PERIODIC) acc_d.outflow -= (double)Hxm.x;
        if (x == n - 1 && p.bc[1] != EMMA_RT_BC_PERIODIC) acc_d.outflow += (double)Hxp.x;
        if (y == 0 && p.bc[2] != EMMA_RT_BC_PERIODIC) acc_d.outflow -= (double)Hym.x;
        if (y == n - 1 && p.bc[3] != EMMA_RT_BC_PERIODIC) acc_d.outflow += (double)Hyp.x;
        if (z == 0 && p.bc[4] != EMMA_RT_BC_PERIODIC) acc_d.outflow -= (double)Hz_lo;
        if (z == n - 1 && p.bc[5] != EMMA_RT_BC_PERIODIC) acc_d.outflow += (double)Hzp.x;
      }
    }
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
