// fused.cu -- single-pass coupled step on the unrefined coarse cells: M1 transport and
// the first trip of the thermo-chemistry sub-cycle loop (rows a-3, a-4) in ONE kernel, so that the radiation field
// crosses HBM once per step (SURVEY.md 8(d) "fused transport -> chemistry", 8(f) NEXT-3):
//
//     unfused: transport 16G + 16G B, chemistry 16G + 12 + 16G + 8 B          = 64 G + 20 B per cell  (212 B at G = 3)
//     fused:   read U 16G, n0, x, e 12; write U 16G, x, e 8                   = 32 G + 20 B per cell  (116 B at G = 3)
//
// Legal because transport is a Jacobi update (reads only the old buffer, Eq. 30) and the chemistry
// of Eq. 43-48 is cell-local.  The arithmetic is that of transport_tma.cu followed by that of
// chem_main_kernel (chem_math.cuh): a cell whose first chemical time guess covers the whole step and whose attempt
// passes the 10 % rule is finished here; every other unrefined cell is written with its post-transport radiation
// U* and appended to the queue of chem_tail_kernel; a refined coarse cell is written with U* for the CRTA kernels.
//
// Shape: a CTA of 512 threads owns a 32 x 16 column (one cell per thread) and marches along z; ALL G groups of a
// plane sit in one stage of a TMA-fed shared-memory ring (cp.async.bulk.tensor boxes completing on mbarriers), so a
// thread has the G post-transport values of its cell in registers when the chemistry starts.  The ring keeps
// planes j-1, j, j+1 (the z-neighbours are read from shared memory, not carried in registers: there are G of them)
// plus NST-3 planes in flight.  Closures (a, b) are computed once per cell when its plane lands and staged in a
// pair of closure planes (plane j's, and plane j-1's whose slots receive plane j+1's as they are consumed); one
// __syncthreads per plane.
#include <cuda.h>

#include "async_copy.cuh"
#include "chem_math.cuh"
#include "emma_rt_internal.cuh"
#include "transport_math.cuh"

namespace emma {

namespace {

using namespace acp;

constexpr int TX = 32;                         // tile width = one warp along x
#ifndef FUSED_TY
#define FUSED_TY 16
#endif
constexpr int TY = FUSED_TY;                   // tile height = warps per CTA.  16: one CTA of 512 threads per SM (3.95 ms
                                               // at 512^3 x 3); 8: two CTAs of 256 (measured slower: 4.19 ms, more halo work)
constexpr int CTAS_PER_SM = 16 / TY;
constexpr int NT = TX * TY;
constexpr int ROWB = TX * 16;                  // bytes of one row of cells
constexpr int TOPROW = (TY + 1) * ROWB;        // offset of the y-halo row above
constexpr int STAGE_ROWS = (TY + 2) * ROWB;    // rows region of one group's plane
constexpr int COLB = TY * 16;                  // bytes of one halo column
constexpr int SG = STAGE_ROWS + 2 * COLB;      // one group's plane: what its five boxes deliver
constexpr int ABG = SG / 2;                    // its closure plane: float2 (a, b) at half the byte offset of the cell

template <int G> constexpr int fused_nst() { return TY == 16 ? (G == 1 ? 12 : G == 2 ? 8 : G == 3 ? 6 : 4) : (G == 1 ? 10 : G == 2 ? 7 : G == 3 ? 5 : 4); }
template <int G> constexpr size_t fused_smem() { return (size_t)fused_nst<G>() * G * SG + 2 * G * ABG + 8 * (fused_nst<G>() + 1); }

template <int G, bool BCGEN>
__global__ void __launch_bounds__(NT, CTAS_PER_SM)
fused_kernel(const TransportParams p, const __grid_constant__ TransportMaps maps, float4* __restrict__ Uout,
             const ChemParams cp, const LevelDev L, int* __restrict__ queue, unsigned int* __restrict__ qcount,
             Partial* __restrict__ parts)
{
  constexpr int NST = fused_nst<G>();
  constexpr int STAGE = G * SG, ABP = G * ABG;
  extern __shared__ __align__(128) unsigned char smem[];
  unsigned char* const sAB = smem + NST * STAGE;
  const unsigned bar0 = smem_u32(sAB + 2 * ABP);
  const unsigned stage0 = smem_u32(smem);
  // "plane done" barrier: a warp arrives when its reads of planes j-1 / j and its closure writes of plane j+1 are
  // complete; everyone waits for it at the top of the next plane (split-phase: the chemistry runs in between, so the
  // warps do not have to finish a plane together)
  const unsigned bar_pl = bar0 + 8 * NST;

  const int n = p.n;
  int bid = blockIdx.x;
  const int tix = bid % p.tiles_x; bid /= p.tiles_x;
  const int tiy = bid % p.tiles_y; bid /= p.tiles_y;
  const int izc = bid;
  const int x0 = tix * TX, y0 = tiy * TY;
  const int wx = min(TX, n - x0), wy = min(TY, n - y0);
  const int z0 = p.z_lo + izc * p.zchunk, z1 = min(p.z_hi, z0 + p.zchunk);
  const int zc = z1 - z0;
  const int t = threadIdx.x, lane = t & 31;
  const int tx = t % TX, ty = t / TX;
  const int x = x0 + tx, y = y0 + ty;
  const bool act = (tx < wx) && (ty < wy);

  // neighbours inside a group's plane (byte offsets)
  const int own = (ty + 1) * ROWB + tx * 16;
  const int oxm = (tx > 0) ? own - 16 : STAGE_ROWS + ty * 16;
  const int oxp = (tx < wx - 1) ? own + 16 : STAGE_ROWS + COLB + ty * 16;
  const int oym = own - ROWB;
  const int oyp = (ty + 1 < wy) ? own + ROWB : TOPROW + tx * 16;
  // halo closures: the 2 wy + 2 wx halo cells of each of the G groups are dealt in order, task h -> thread h: whole
  // warps (288 tasks = 9 of the 16 warps at G = 3) so that the others skip the work altogether, and consecutive lanes
  // read consecutive cells (no bank conflicts).  The split-phase plane barrier lets the lighter warps run ahead.
  // (with 32 x 8 tiles and G = 4 there are more halo cells than threads: a second task for some)
  auto halo_task = [&](int h) -> int {         // byte offset (inside a stage) of halo task h, or -1
    const int nh = 2 * wy + 2 * wx;
    if (h >= nh * G) return -1;
    const int g = h / nh, q = h - g * nh;
    const int o = (q < wy) ? STAGE_ROWS + q * 16 : (q < 2 * wy) ? STAGE_ROWS + COLB + (q - wy) * 16
                : (q < 2 * wy + wx) ? (q - 2 * wy) * 16 : TOPROW + (q - 2 * wy - wx) * 16;
    return g * SG + o;
  };
  const int hoff = halo_task(t);
  const int hoff2 = ((2 * TY + 2 * TX) * G > NT) ? halo_task(NT + t) : -1;
  float sxm = 1.f, sxp = 1.f, sym = 1.f, syp = 1.f;     // reflective faces: sign of the face-normal flux (A13)
  if (BCGEN) {
    if (tx == 0 && x0 == 0 && p.bc[0] == EMMA_RT_BC_REFLECTIVE) sxm = -1.f;
    if (tx == wx - 1 && x0 + wx == n && p.bc[1] == EMMA_RT_BC_REFLECTIVE) sxp = -1.f;
    if (ty == 0 && y0 == 0 && p.bc[2] == EMMA_RT_BC_REFLECTIVE) sym = -1.f;
    if (ty == wy - 1 && y0 + wy == n && p.bc[3] == EMMA_RT_BC_REFLECTIVE) syp = -1.f;
  }

  bool flz, fltop, fl;
  const int zm = bc_map(z0 - 1, n, p.bc[4], p.bc[5], flz);
  const int ztop = bc_map(z1, n, p.bc[4], p.bc[5], fltop);
  const int cxl = 4 * bc_map(x0 - 1, n, p.bc[0], p.bc[1], fl);
  const int cxr = 4 * bc_map(x0 + wx, n, p.bc[0], p.bc[1], fl);
  const int cyb = bc_map(y0 - 1, n, p.bc[2], p.bc[3], fl);
  const int cyt = bc_map(y0 + wy, n, p.bc[2], p.bc[3], fl);

  // plane j (relative to z0; -1 = the plane below, zc = the plane above), all G groups -> stage s.  The 5 G boxes of a
  // plane are issued by the first lanes of 5 G different warps (each arrives on the stage's mbarrier with its own
  // byte count), so that no single warp carries the whole descriptor traffic on the critical path of the plane loop.
  const int warp = t >> 5;
  auto issue = [&](int j, int s) {
    if (lane != 0) return;
    const int zz = (j < 0) ? zm : (j >= zc) ? ztop : z0 + j;
    const unsigned bar = bar0 + 8 * s;
    for (int b = warp; b < 5 * G; b += NT / 32) {
      const int g = b / 5, k = b - 5 * g;
      const unsigned dst = stage0 + s * STAGE + g * SG;
      const int zg = g * n + zz;
      if (k == 0) { mbar_expect_tx(bar, TY * ROWB); tma_load_3d(dst + ROWB, &maps.main, bar, 4 * x0, y0, zg); }
      else if (k == 1) { mbar_expect_tx(bar, ROWB); tma_load_3d(dst, &maps.row, bar, 4 * x0, cyb, zg); }
      else if (k == 2) { mbar_expect_tx(bar, ROWB); tma_load_3d(dst + TOPROW, &maps.row, bar, 4 * x0, cyt, zg); }
      else if (k == 3) { mbar_expect_tx(bar, COLB); tma_load_3d(dst + STAGE_ROWS, &maps.col, bar, cxl, y0, zg); }
      else { mbar_expect_tx(bar, COLB); tma_load_3d(dst + STAGE_ROWS + COLB, &maps.col, bar, cxr, y0, zg); }
    }
  };

  if (t == 0) {
    for (int s = 0; s < NST; s++) mbar_init(bar0 + 8 * s, 5 * G);
    mbar_init(bar_pl, NT / 32);
    mbar_fence_init();
  }
  __syncthreads();
  for (int j = -1; j < NST - 1 && j <= zc; j++) issue(j, j + 1);

  const float c0 = p.c0, c1 = p.c1;
  const size_t plane = (size_t)n * n, ncell = plane * n;
  Acc acc_d;
  double t_abs = 0.0, t_tot = 0.0, t_inj = 0.0, t_rec = 0.0;          // fast-path tallies, per unit volume
  unsigned n_fast = 0;                                               // cells finished here (one accepted sub-step each)

  // closures of plane in stage `st` into closure plane `ab`: my own cell (all groups) and my halo cell
  auto stage_closures = [&](const unsigned char* st, unsigned char* ab, bool halo) {
#pragma unroll
    for (int g = 0; g < G; g++) {
      float a, b;
      closure_ab(*(const float4*)(st + g * SG + own), a, b);
      *(float2*)(ab + g * ABG + (own >> 1)) = make_float2(a, b);
    }
    if (halo && hoff >= 0) {
      float a, b;
      closure_ab(*(const float4*)(st + hoff), a, b);
      *(float2*)(ab + (hoff >> 1)) = make_float2(a, b);
    }
    if (halo && hoff2 >= 0) {
      float a, b;
      closure_ab(*(const float4*)(st + hoff2), a, b);
      *(float2*)(ab + (hoff2 >> 1)) = make_float2(a, b);
    }
  };

  // ---- prologue: closures of plane -1 (own cells only: it is only ever a z-neighbour) and of plane 0
  mbar_wait(bar0, 0);
  stage_closures(smem, sAB, false);
  mbar_wait(bar0 + 8, 0);
  stage_closures(smem + STAGE, sAB + ABP, true);
  __syncthreads();

  int s_old = 0, s_blw = 0, s_cur = 1, s_nxt = 2 % NST;   // stages of planes j-2 (free), j-1, j, j+1
  unsigned par_nxt = (2 / NST) & 1;            // phase parity of plane j+1's stage
  int ab_blw = 0, ab_cur = 1;                  // closure planes of j-1 (reused for j+1) and j

  unsigned pend_m = 0, pend_b = 0;             // deferred cells of the previous plane: ballot, queue base (in flight)
  int pend_cell = 0;
  auto flush_deferred = [&]() {
    if (pend_m) {
      const unsigned b = __shfl_sync(0xffffffffu, pend_b, __ffs(pend_m) - 1);
      if ((pend_m >> lane) & 1u) queue[b + __popc(pend_m & ((1u << lane) - 1u))] = pend_cell;
    }
  };

  // my cell of plane j, advanced by one plane per trip: 32 bits (n <= 1290, checked at init), so that an array element's
  // address is one IMAD.WIDE
  const unsigned plane32 = (unsigned)n * (unsigned)n;
  unsigned cell = (unsigned)z0 * plane32 + (act ? (unsigned)y * (unsigned)n + (unsigned)x : 0u);
  for (int j = 0; j < zc; j++, cell += plane32) {
    const int z = z0 + j;
    // chemistry inputs of my cell: in flight while the transport arithmetic runs
    float n0v = 1.f, xsv = 0.f, epsv = 1.f;
    unsigned srcw = 0;
    bool chem = act;
    if (act) {
      n0v = L.n0[cell]; xsv = L.xs[cell]; epsv = L.eps[cell];
      if (L.n_src) srcw = L.srcmask[cell >> 5];
      if (L.refined) chem = !((L.refined[cell >> 5] >> (cell & 31)) & 1u);            // split cells: CRTA kernels
    }
    if (j > 0) {
      // every warp is done with plane j-2's stage and with the closure plane that now receives plane j+1
      mbar_wait_relaxed(bar_pl, (unsigned)(j - 1) & 1u);
      if (j + NST - 2 <= zc) issue(j + NST - 2, s_old);
    }
    const unsigned char* sb = smem + s_blw * STAGE;
    const unsigned char* sc = smem + s_cur * STAGE;
    const unsigned char* sn = smem + s_nxt * STAGE;
    unsigned char* ABb = sAB + ab_blw * ABP;                           // closures of plane j-1; receives plane j+1
    const unsigned char* ABc = sAB + ab_cur * ABP;
    mbar_wait(bar0 + 8 * s_nxt, par_nxt);
    const bool top = (j + 1 == zc);

    CellState<G> c;
#pragma unroll
    for (int g = 0; g < G; g++) {
      // z-neighbours: same (x, y) in the stages of planes j-1 and j+1
      float4 ub = *(const float4*)(sb + g * SG + own);
      const float2 abb = *(const float2*)(ABb + g * ABG + (own >> 1));
      float4 un = *(const float4*)(sn + g * SG + own);
      if (BCGEN) {
        if (j == 0 && flz) ub.w = -ub.w;
        if (top && fltop) un.w = -un.w;
      }
      float na, nb;
      closure_ab(un, na, nb);
      if (!top) *(float2*)(ABb + g * ABG + (own >> 1)) = make_float2(na, nb);
      float4 acc = below_z(ub, abb.x, abb.y);
      add_plus<2>(acc, un, na, nb);
      // x / y neighbours from the stage of plane j and its closure plane
      const unsigned char* scg = sc + g * SG;
      const unsigned char* abg = ABc + g * ABG;
      float4 u; float2 ab;
      u = *(const float4*)(scg + oxm); ab = *(const float2*)(abg + (oxm >> 1)); if (BCGEN) u.y *= sxm; add_minus<0>(acc, u, ab.x, ab.y);
      u = *(const float4*)(scg + oxp); ab = *(const float2*)(abg + (oxp >> 1)); if (BCGEN) u.y *= sxp; add_plus<0>(acc, u, ab.x, ab.y);
      u = *(const float4*)(scg + oym); ab = *(const float2*)(abg + (oym >> 1)); if (BCGEN) u.z *= sym; add_minus<1>(acc, u, ab.x, ab.y);
      u = *(const float4*)(scg + oyp); ab = *(const float2*)(abg + (oyp >> 1)); if (BCGEN) u.z *= syp; add_plus<1>(acc, u, ab.x, ab.y);
      const float4 cu = *(const float4*)(scg + own);
      float4 o;
      mul2(o.x, o.y, cu.x, cu.y, c0, c0); mul2(o.z, o.w, cu.z, cu.w, c0, c0);
      fma2(o.x, o.y, acc.x, acc.y, c1, c1, o.x, o.y); fma2(o.z, o.w, acc.z, acc.w, c1, c1, o.z, o.w);
      c.N[g] = o.x; c.px[g] = o.y; c.py[g] = o.z; c.pz[g] = o.w;
      if (BCGEN && act) {
        // outflow through open faces (A15): transmissive face flux = own F_d (ghost copies the cell), reflective = 0
        if (x == 0 && p.bc[0] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cu.y;
        if (x == n - 1 && p.bc[1] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cu.y;
        if (y == 0 && p.bc[2] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cu.z;
        if (y == n - 1 && p.bc[3] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cu.z;
        if (z == 0 && p.bc[4] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cu.w;
        if (z == n - 1 && p.bc[5] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cu.w;
      }
    }

    if (!top && hoff >= 0) {                   // my halo cell of plane j+1 (read by others one plane later)
      float a, b;
      closure_ab(*(const float4*)(sn + hoff), a, b);
      *(float2*)(ABb + (hoff >> 1)) = make_float2(a, b);
    }
    if (!top && hoff2 >= 0) {
      float a, b;
      closure_ab(*(const float4*)(sn + hoff2), a, b);
      *(float2*)(ABb + (hoff2 >> 1)) = make_float2(a, b);
    }
    // my part of planes j-1, j, j+1 is done (release: the closure writes above)
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_pl);

    // ---- chemistry: the first trip of the sub-cycle loop when it covers the whole step (as chem_main_kernel)
    bool defer = false;
    if (act) {
      bool go = chem;
      Rates r;
      float dmin = FINF;
      if (chem) {
        c.n0 = n0v; c.eps = epsv;
        decode_x(xsv, c.x, c.y);
        load_sources_word<G>(L, (long long)cell, srcw, c.S);
        const float T = c.eps * frcp(KB15 * (1.f + c.x));
        r = rates_at(T, cp.otsa, c.x, c.n0);
        if (cp.thermal) {
          float hsum = 0.f;
#pragma unroll
          for (int g = 0; g < G; g++) hsum = fmaf(cp.csigE[g], c.N[g], hsum);
          const float d = c.y * hsum - c.n0 * c.x * fmaf(c.y, r.cHI, c.x * r.cHII);
          const float guess = first_guess(c.eps, d, cp.dt);                    // PAPER.md:290 (A9)
          go = guess >= cp.dt;
          if (go) dmin = guess;
        }
      }
      float N1[G], iden[G], x1, y1, eps1;
      if (go) go = attempt<G>(cp, c, r, cp.dt, N1, iden, x1, y1, eps1);
      if (go) {
        // commit.  The tallies of A15 are summed per thread in fp64 and scaled by the (one) cell volume at the end;
        // the injected term exists in source cells only, the recombination term without OTSA only.
        CellTally tl;
        const float k = c.y * c.n0 * cp.dt;
        float sumN = 0.f;
#pragma unroll
        for (int g = 0; g < G; g++) {
          tl.absorbed = fmaf(cp.csig[g] * k, N1[g], tl.absorbed);
          c.N[g] = N1[g];
          sumN += N1[g];
          c.px[g] = decay(c.px[g], iden[g]); c.py[g] = decay(c.py[g], iden[g]); c.pz[g] = decay(c.pz[g], iden[g]);
        }
        c.x = x1; c.y = y1; c.eps = eps1;
        tl.nsub = 1;
        store_cell<G>(L, (long long)cell, Uout, (long long)ncell, c, tl, cp.record);
        t_abs += (double)tl.absorbed;
        t_tot += (double)sumN;
        // S is 0 outside source cells and r.rec is 0 with OTSA: adding +0.0 leaves the sums as they are, without the predicates
        float inj = 0.f;
#pragma unroll
        for (int g = 0; g < G; g++) inj = fmaf(c.S[g], cp.dt, inj);
        t_inj += (double)inj;
        t_rec += (double)(r.rec * cp.dt);
        n_fast++;
        acc_d.dtau_min = fminf(acc_d.dtau_min, dmin);
        if (!finite_cell<G>(c)) acc_d.nonfinite++;
      } else {
        // post-transport radiation only: the tail kernel (deferred) or the CRTA kernels (split cell) take it from here
#pragma unroll
        for (int g = 0; g < G; g++) Uout[(size_t)g * ncell + cell] = make_float4(c.N[g], c.px[g], c.py[g], c.pz[g]);
        defer = chem;
      }
    }
    // warp-aggregated append of the deferred cells (north_star item 3: warp-level work compaction).  The atomic that
    // reserves the queue slots is issued here and its result consumed one plane later, off the critical path.
    flush_deferred();
    pend_m = __ballot_sync(0xffffffffu, defer);
    if (pend_m) {
      if (lane == __ffs(pend_m) - 1) pend_b = atomicAdd(qcount, (unsigned)__popc(pend_m));
      pend_cell = (int)cell;
      if (defer) acc_d.ndefer++;
    }

    s_old = s_blw; s_blw = s_cur; s_cur = s_nxt;
    if (++s_nxt == NST) { s_nxt = 0; par_nxt ^= 1u; }
    const int ab_nxt = ab_blw;
    ab_blw = ab_cur; ab_cur = ab_nxt;
  }
  flush_deferred();

  acc_d.absorbed = t_abs * L.dV; acc_d.injected = t_inj * L.dV; acc_d.recomb = t_rec * L.dV; acc_d.total = t_tot * L.dV_total;
  acc_d.nsub = n_fast; acc_d.nsub_max = n_fast ? 1u : 0u;
  acc_d.outflow *= (double)p.nu * p.dV;
  block_reduce_store(acc_d, parts + blockIdx.x);
}

template <int G>
int launch_G(const TransportParams& p, const TransportMaps& maps, float4* Uout, const ChemParams& cp, const LevelDev& L0,
             int* queue, unsigned int* qcount, Partial* parts, int nblk, bool bcgen, cudaStream_t st)
{
  if (bcgen) fused_kernel<G, true><<<nblk, NT, fused_smem<G>(), st>>>(p, maps, Uout, cp, L0, queue, qcount, parts);
  else fused_kernel<G, false><<<nblk, NT, fused_smem<G>(), st>>>(p, maps, Uout, cp, L0, queue, qcount, parts);
  return 1;
}

template <int G>
cudaError_t configure_G()
{
  cudaError_t e = cudaFuncSetAttribute(fused_kernel<G, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<G>());
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(fused_kernel<G, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<G>());
}

}  // namespace

// Per-device set-up (emma_rt_init, handle's device current): dynamic shared memory opt-in of the kernels for G groups
cudaError_t configure_fused(int G)
{
  switch (G) {
    case 1: return configure_G<1>();
    case 2: return configure_G<2>();
    case 3: return configure_G<3>();
    default: return configure_G<4>();
  }
}

// CTAs resident per SM of the fused pass (one: its ring fills the shared memory) -- for the z-chunk cost model
int fused_ctas_per_sm() { return CTAS_PER_SM; }
int fused_tile_y() { return TY; }

// Launches the fused pass over the coarse block; p.tiles_* / p.zchunk / p.nzc describe its own 32 x 16 tiling.
int launch_fused(const TransportParams& p, const TransportMaps& maps_in, float4* Uout, const ChemParams& cp,
                 const LevelDev& L0, int* queue, unsigned int* qcount, Partial* parts, int* n_parts, cudaStream_t st)
{
  const int nblk = p.tiles_x * p.tiles_y * p.nzc;
  bool bcgen = false;
  for (int f = 0; f < 6; f++) bcgen = bcgen || (p.bc[f] != EMMA_RT_BC_PERIODIC);
  int k;
  switch (p.G) {
    case 1: k = launch_G<1>(p, maps_in, Uout, cp, L0, queue, qcount, parts, nblk, bcgen, st); break;
    case 2: k = launch_G<2>(p, maps_in, Uout, cp, L0, queue, qcount, parts, nblk, bcgen, st); break;
    case 3: k = launch_G<3>(p, maps_in, Uout, cp, L0, queue, qcount, parts, nblk, bcgen, st); break;
    default: k = launch_G<4>(p, maps_in, Uout, cp, L0, queue, qcount, parts, nblk, bcgen, st); break;
  }
  *n_parts = k ? nblk : 0;
  return k;
}

}  // namespace emma
