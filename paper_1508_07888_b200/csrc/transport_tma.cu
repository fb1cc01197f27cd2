// transport_tma.cu -- explicit M1 transport on the coarse block, TMA-fed.
//
// Same arithmetic as transport.cu (Eq. 30 + 32 with the closure Eq. 22-23, readings A1-A4, A13);
// what changes is how the planes reach the SM.  transport.cu holds the planes in flight in registers (one plane
// ahead: ~25 KB per SM) and is bound by memory-level parallelism (profiles/r1b_summary.md: 38 % issue slots,
// long-scoreboard stalls, 49 % DRAM).  Here one thread per CTA feeds a ring of NST shared-memory stages with
// cp.async.bulk.tensor (TMA) loads that complete on mbarriers, NST-2 planes ahead of the march, at no register cost:
//
//   stage = [18 rows x 32 cells]  rows 1..16: the tile's own cells (one 32 x 16 box)
//                                 row 0 / row 17: the y-halo rows below / above (two 32 x 1 boxes)
//           [Lcol 16][Rcol 16]    the x-halo columns (two 1 x 16 boxes)
//
// Every box is addressed by tensor coordinates, so the boundary conditions of PAPER.md:436 are coordinate maps of
// the halo boxes (periodic: wrapped coordinate; transmissive / reflective: the tile's own edge, the reflective sign
// applied by the consumer); cells outside a ragged tile are zero-filled by the TMA unit.  The z-neighbours of a
// thread's two cells stay in registers (CUR / NXT / the folded plane below), the x/y-neighbours and their closures
// (a, b), computed once per cell and staged in a double-buffered closure plane, come from shared memory; one
// __syncthreads per plane.
#include <cuda.h>

#include "async_copy.cuh"
#include "emma_rt_internal.cuh"
#include "transport_math.cuh"

namespace emma {

namespace {

constexpr int TX = 32;                         // tile width = one warp along x
constexpr int TYT = 8;                         // thread rows
constexpr int CY = 2;                          // cells per thread along y
constexpr int TY = TYT * CY;
constexpr int NT = TX * TYT;
constexpr int ROWB = TX * 16;                  // bytes of one row of cells
constexpr int TOPROW = (TY + 1) * ROWB;        // offset of the y-halo row above
constexpr int STAGE_ROWS = (TY + 2) * ROWB;    // rows region of a stage
constexpr int COLB = TY * 16;                  // bytes of one halo column
constexpr int STAGE_BYTES = STAGE_ROWS + 2 * COLB;     // = bytes one plane's five boxes deliver
constexpr int AB_BYTES = STAGE_BYTES / 2;      // closure plane: float2 (a, b) at half the byte offset of the cell

using namespace acp;

struct TileT {                                 // per-thread constants of the march
  int own0;                                    // byte offset of my first cell inside a stage (second = own0 + ROWB)
  int xm0, xp0, xm1, xp1, ym0, yp0, yp1;       // neighbours that come from shared memory
  int hoff;                                    // halo cell whose closure I compute (or -1)
  bool act0, act1, pair;
  float sxm, sxp, sym, syp;                    // reflective faces: sign of the face-normal flux of that neighbour (A13)
};

}  // namespace

// NST: stages of the ring.  DIAG / BCGEN as in transport.cu (BCGEN: some face is not periodic -> outflow sums and the
// reflective signs are compiled in).
template <int NST, bool DIAG, bool BCGEN>
__global__ void __launch_bounds__(NT, 2)
transport_tma_kernel(const TransportParams p, const __grid_constant__ TransportMaps maps,
                     float4* __restrict__ Uout, Partial* __restrict__ parts)
{
  extern __shared__ __align__(128) unsigned char smem[];
  unsigned char* const sAB = smem + NST * STAGE_BYTES;
  const unsigned bar0 = smem_u32(smem + NST * STAGE_BYTES + 2 * AB_BYTES);
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
  const int t = threadIdx.x;
  const int tx = t % TX, ly = CY * (t / TX);
  const int x = x0 + tx, y = y0 + ly;

  TileT T;
  T.pair = ly + 1 < wy;
  T.act0 = (tx < wx) && (ly < wy);
  T.act1 = (tx < wx) && T.pair;
  T.own0 = (ly + 1) * ROWB + tx * 16;
  const int own1 = T.own0 + ROWB;
  T.xm0 = (tx > 0) ? T.own0 - 16 : STAGE_ROWS + ly * 16;
  T.xm1 = (tx > 0) ? own1 - 16 : STAGE_ROWS + (ly + 1) * 16;
  T.xp0 = (tx < wx - 1) ? T.own0 + 16 : STAGE_ROWS + COLB + ly * 16;
  T.xp1 = (tx < wx - 1) ? own1 + 16 : STAGE_ROWS + COLB + (ly + 1) * 16;
  T.ym0 = T.own0 - ROWB;
  T.yp0 = TOPROW + tx * 16;                    // used only when my second row is outside the tile
  T.yp1 = (ly + 2 < wy) ? own1 + ROWB : TOPROW + tx * 16;
  T.hoff = -1;
  if (t < 2 * wy) T.hoff = STAGE_ROWS + ((t < wy) ? t * 16 : COLB + (t - wy) * 16);
  else if (t < 2 * wy + 2 * wx) { const int q = t - 2 * wy; T.hoff = (q < wx) ? q * 16 : TOPROW + (q - wx) * 16; }
  T.sxm = T.sxp = T.sym = T.syp = 1.f;
  if (BCGEN) {
    if (tx == 0 && x0 == 0 && p.bc[0] == EMMA_RT_BC_REFLECTIVE) T.sxm = -1.f;
    if (tx == wx - 1 && x0 + wx == n && p.bc[1] == EMMA_RT_BC_REFLECTIVE) T.sxp = -1.f;
    if (ly == 0 && y0 == 0 && p.bc[2] == EMMA_RT_BC_REFLECTIVE) T.sym = -1.f;
    if ((T.pair ? ly + 1 : ly) == wy - 1 && y0 + wy == n && p.bc[3] == EMMA_RT_BC_REFLECTIVE) T.syp = -1.f;
  }

  bool flz, fltop, fl;
  const int zm = bc_map(z0 - 1, n, p.bc[4], p.bc[5], flz);
  const int ztop = bc_map(z1, n, p.bc[4], p.bc[5], fltop);
  // halo box coordinates (x in floats)
  const int cxl = 4 * bc_map(x0 - 1, n, p.bc[0], p.bc[1], fl);
  const int cxr = 4 * bc_map(x0 + wx, n, p.bc[0], p.bc[1], fl);
  const int cyb = bc_map(y0 - 1, n, p.bc[2], p.bc[3], fl);
  const int cyt = bc_map(y0 + wy, n, p.bc[2], p.bc[3], fl);
  const int zbase = g * n;

  // plane j (relative to z0; -1 = the plane below, zc = the plane above) -> stage s
  auto issue = [&](int j, int s) {
    const int zz = zbase + ((j < 0) ? zm : (j >= zc) ? ztop : z0 + j);
    const unsigned dst = stage0 + s * STAGE_BYTES, bar = bar0 + 8 * s;
    mbar_expect_tx(bar, STAGE_BYTES);
    tma_load_3d(dst + ROWB, &maps.main, bar, 4 * x0, y0, zz);
    tma_load_3d(dst, &maps.row, bar, 4 * x0, cyb, zz);
    tma_load_3d(dst + TOPROW, &maps.row, bar, 4 * x0, cyt, zz);
    tma_load_3d(dst + STAGE_ROWS, &maps.col, bar, cxl, y0, zz);
    tma_load_3d(dst + STAGE_ROWS + COLB, &maps.col, bar, cxr, y0, zz);
  };

  if (t == 0) {
    for (int s = 0; s < NST; s++) mbar_init(bar0 + 8 * s, 1);
    mbar_fence_init();
  }
  __syncthreads();
  if (t == 0) {
    for (int j = -1; j < NST - 1 && j <= zc; j++) issue(j, j + 1);
  }

  const float c0 = p.c0, c1 = p.c1;
  Acc acc_d;
  float4* pst = Uout + ((size_t)g * n + z0) * n * n + (T.act0 ? ((size_t)y * n + x) : 0);
  const size_t plane = (size_t)n * n;
  const ptrdiff_t d1 = T.act1 ? n : 0;

  // closure of my halo cell of the plane in stage `st`, into closure buffer `ab`
  auto halo_closure = [&](const unsigned char* st, unsigned char* ab) {
    if (T.hoff >= 0) {
      const float4 h = *(const float4*)(st + T.hoff);
      float a, b;
      closure_ab(h, a, b);
      *(float2*)(ab + (T.hoff >> 1)) = make_float2(a, b);
    }
  };

  // ---- prologue: plane -1 folds into W, plane 0 becomes CUR
  float4 W0, W1, cu0, cu1, nu0, nu1;
  float ca0, cb0, ca1, cb1, na0, nb0, na1, nb1;
  {
    mbar_wait(bar0, 0);
    float4 m0 = *(const float4*)(smem + T.own0), m1 = *(const float4*)(smem + own1);
    if (flz) { m0.w = -m0.w; m1.w = -m1.w; }
    float a, b;
    closure_ab(m0, a, b); W0 = below_z(m0, a, b);
    closure_ab(m1, a, b); W1 = below_z(m1, a, b);
    mbar_wait(bar0 + 8, 0);
    const unsigned char* st = smem + STAGE_BYTES;
    cu0 = *(const float4*)(st + T.own0); cu1 = *(const float4*)(st + own1);
    closure_ab(cu0, ca0, cb0); closure_ab(cu1, ca1, cb1);
    *(float2*)(sAB + (T.own0 >> 1)) = make_float2(ca0, cb0);
    *(float2*)(sAB + (own1 >> 1)) = make_float2(ca1, cb1);
    halo_closure(st, sAB);
  }
  __syncthreads();
  if (t == 0 && NST - 1 <= zc) issue(NST - 1, 0);

  int s_cur = 1;                               // stage of plane j
  int s_nxt = (2 % NST);                       // stage of plane j + 1
  unsigned par_nxt = (2 / NST) & 1;            // its phase parity
  int j = 0;

  // one plane: (cu, ca, cb) is plane j, (nu, na, nb) receives plane j + 1; ABC / ABN are the closure buffers of j / j+1
  auto body = [&](float4& cu0, float4& cu1, float& ca0, float& cb0, float& ca1, float& cb1,
                  float4& nu0, float4& nu1, float& na0, float& nb0, float& na1, float& nb1,
                  const unsigned char* ABC, unsigned char* ABN) {
    const unsigned char* sc = smem + s_cur * STAGE_BYTES;
    const unsigned char* sn = smem + s_nxt * STAGE_BYTES;
    // (a) plane j + 1 has landed: my two cells, their closure; stage the closures for the next iteration
    mbar_wait(bar0 + 8 * s_nxt, par_nxt);
    nu0 = *(const float4*)(sn + T.own0); nu1 = *(const float4*)(sn + own1);
    const bool top = (j + 1 == zc);
    if (top && fltop) { nu0.w = -nu0.w; nu1.w = -nu1.w; }
    closure_ab(nu0, na0, nb0); closure_ab(nu1, na1, nb1);
    if (!top) {
      *(float2*)(ABN + (T.own0 >> 1)) = make_float2(na0, nb0);
      *(float2*)(ABN + (own1 >> 1)) = make_float2(na1, nb1);
      halo_closure(sn, ABN);
    }
    // (b) z-neighbours and the y-neighbour inside the pair, all in registers
    float4 acc0 = W0, acc1 = W1;
    add_plus<2>(acc0, nu0, na0, nb0);
    add_plus<2>(acc1, nu1, na1, nb1);
    if (T.pair) add_plus<1>(acc0, cu1, ca1, cb1);
    add_minus<1>(acc1, cu0, ca0, cb0);
    // (c) the other x / y neighbours from the stage of plane j and its closure plane
    auto nb_load = [&](int off, float4& u, float2& ab) {
      u = *(const float4*)(sc + off);
      ab = *(const float2*)(ABC + (off >> 1));
    };
    float4 u; float2 ab;
    if (!T.pair) { nb_load(T.yp0, u, ab); if (BCGEN) u.z *= T.syp; add_plus<1>(acc0, u, ab.x, ab.y); }
    nb_load(T.xm0, u, ab); if (BCGEN) u.y *= T.sxm; add_minus<0>(acc0, u, ab.x, ab.y);
    nb_load(T.xp0, u, ab); if (BCGEN) u.y *= T.sxp; add_plus<0>(acc0, u, ab.x, ab.y);
    nb_load(T.ym0, u, ab); if (BCGEN) u.z *= T.sym; add_minus<1>(acc0, u, ab.x, ab.y);
    nb_load(T.xm1, u, ab); if (BCGEN) u.y *= T.sxm; add_minus<0>(acc1, u, ab.x, ab.y);
    nb_load(T.xp1, u, ab); if (BCGEN) u.y *= T.sxp; add_plus<0>(acc1, u, ab.x, ab.y);
    nb_load(T.yp1, u, ab); if (BCGEN) u.z *= (T.pair ? T.syp : 1.f); add_plus<1>(acc1, u, ab.x, ab.y);
    float4 o0, o1;
    mul2(o0.x, o0.y, cu0.x, cu0.y, c0, c0); mul2(o0.z, o0.w, cu0.z, cu0.w, c0, c0);
    mul2(o1.x, o1.y, cu1.x, cu1.y, c0, c0); mul2(o1.z, o1.w, cu1.z, cu1.w, c0, c0);
    fma2(o0.x, o0.y, acc0.x, acc0.y, c1, c1, o0.x, o0.y); fma2(o0.z, o0.w, acc0.z, acc0.w, c1, c1, o0.z, o0.w);
    fma2(o1.x, o1.y, acc1.x, acc1.y, c1, c1, o1.x, o1.y); fma2(o1.z, o1.w, acc1.z, acc1.w, c1, c1, o1.z, o1.w);
    if (T.act0) pst[0] = o0;
    if (T.act1) pst[d1] = o1;
    if (DIAG) {
      if (T.act0) {
        if (!(fabsf(o0.x) + fabsf(o0.y) + fabsf(o0.z) + fabsf(o0.w) < __int_as_float(0x7f800000))) acc_d.nonfinite++;
        acc_d.total += (double)o0.x;
      }
      if (T.act1) {
        if (!(fabsf(o1.x) + fabsf(o1.y) + fabsf(o1.z) + fabsf(o1.w) < __int_as_float(0x7f800000))) acc_d.nonfinite++;
        acc_d.total += (double)o1.x;
      }
    }
    if (BCGEN) {
      // outflow through open faces (A15): transmissive face flux = own F_d (ghost copies the cell), reflective = 0
      const int z = z0 + j;
      if (T.act0) {
        if (x == 0 && p.bc[0] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cu0.y;
        if (x == n - 1 && p.bc[1] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cu0.y;
        if (y == 0 && p.bc[2] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cu0.z;
        if (y == n - 1 && p.bc[3] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cu0.z;
        if (z == 0 && p.bc[4] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cu0.w;
        if (z == n - 1 && p.bc[5] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cu0.w;
      }
      if (T.act1) {
        if (x == 0 && p.bc[0] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cu1.y;
        if (x == n - 1 && p.bc[1] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cu1.y;
        if (y + 1 == n - 1 && p.bc[3] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cu1.z;
        if (z == 0 && p.bc[4] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cu1.w;
        if (z == n - 1 && p.bc[5] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cu1.w;
      }
    }
    // (d) this plane becomes the one below; its stage is free once every thread has passed the barrier
    W0 = below_z(cu0, ca0, cb0);
    W1 = below_z(cu1, ca1, cb1);
    __syncthreads();
    if (t == 0 && j + NST <= zc) issue(j + NST, s_cur);
    s_cur = s_nxt;
    if (++s_nxt == NST) { s_nxt = 0; par_nxt ^= 1u; }
    pst += plane;
    j++;
  };

  unsigned char* const AB0 = sAB;
  unsigned char* const AB1 = sAB + AB_BYTES;
  for (;;) {
    body(cu0, cu1, ca0, cb0, ca1, cb1, nu0, nu1, na0, nb0, na1, nb1, AB0, AB1); if (j >= zc) break;
    body(nu0, nu1, na0, nb0, na1, nb1, cu0, cu1, ca0, cb0, ca1, cb1, AB1, AB0); if (j >= zc) break;
  }

  if (DIAG || BCGEN) {
    acc_d.outflow *= (double)p.nu * p.dV;
    acc_d.total *= p.dV;
    block_reduce_store(acc_d, parts + blockIdx.x);
  }
}

// ---- host side ---------------------------------------------------------------------------------------------------

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled()
{
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

constexpr int NST_DEFAULT = 6;

template <int NST>
size_t smem_bytes() { return (size_t)NST * STAGE_BYTES + 2 * AB_BYTES + 8 * NST; }

template <int NST, bool DIAG, bool BCGEN>
cudaError_t launch_variant(const TransportParams& p, const TransportMaps& maps, float4* Uout, Partial* parts, int nblk,
                           cudaStream_t st)
{
  transport_tma_kernel<NST, DIAG, BCGEN><<<nblk, NT, smem_bytes<NST>(), st>>>(p, maps, Uout, parts);
  return cudaSuccess;
}

template <int NST>
cudaError_t launch_nst(const TransportParams& p, const TransportMaps& maps, float4* Uout, Partial* parts, int nblk,
                       bool diag, bool bcgen, cudaStream_t st)
{
  if (diag && bcgen) return launch_variant<NST, true, true>(p, maps, Uout, parts, nblk, st);
  if (diag) return launch_variant<NST, true, false>(p, maps, Uout, parts, nblk, st);
  if (bcgen) return launch_variant<NST, false, true>(p, maps, Uout, parts, nblk, st);
  return launch_variant<NST, false, false>(p, maps, Uout, parts, nblk, st);
}

template <int NST>
cudaError_t configure_nst()
{
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(transport_tma_kernel<NST, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<NST>())) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(transport_tma_kernel<NST, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<NST>())) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(transport_tma_kernel<NST, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<NST>())) != cudaSuccess) return e;
  return cudaFuncSetAttribute(transport_tma_kernel<NST, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<NST>());
}

}  // namespace

// Per-device set-up (emma_rt_init, handle's device current): dynamic shared memory opt-in of every ring depth
cudaError_t configure_transport_tma()
{
  cudaError_t e;
  if ((e = configure_nst<4>()) != cudaSuccess) return e;
  if ((e = configure_nst<NST_DEFAULT>()) != cudaSuccess) return e;
  return configure_nst<8>();
}

// Tensor maps of one radiation buffer U[G][n][n][n] float4, seen as a rank-3 fp32 tensor (4n, n, G n).
// `main_x` > 0: the main box is that many cells wide (a kernel whose rows carry their x halo), the row box stays tile_x wide.
// Returns 0 on success, the CUresult (or -1 when the driver entry point is missing) otherwise.
int make_transport_maps(const float4* U, int n, int G, TransportMaps* out, int tile_y, int tile_x, int main_x)
{
  EncodeTiledFn enc = encode_tiled();
  if (!enc) return -1;
  const cuuint64_t gdim[3] = {(cuuint64_t)4 * n, (cuuint64_t)n, (cuuint64_t)n * G};
  const cuuint64_t gstr[2] = {(cuuint64_t)16 * n, (cuuint64_t)16 * n * n};
  const cuuint32_t estr[3] = {1, 1, 1};
  const cuuint32_t box_main[3] = {4 * (cuuint32_t)(main_x > 0 ? main_x : tile_x), (cuuint32_t)tile_y, 1}, box_row[3] = {4 * (cuuint32_t)tile_x, 1, 1}, box_col[3] = {4, (cuuint32_t)tile_y, 1};
  CUresult r;
  r = enc(&out->main, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)U, gdim, gstr, box_main, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return (int)r;
  r = enc(&out->row, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)U, gdim, gstr, box_row, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return (int)r;
  r = enc(&out->col, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)U, gdim, gstr, box_col, estr,
          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return (int)r;
}

int launch_transport_tma(const TransportParams& p, const TransportMaps& maps_in, float4* Uout, Partial* parts,
                         int* n_parts, cudaStream_t st)
{
  const int nblk = p.tiles_x * p.tiles_y * p.nzc * p.G;
  bool bcgen = false;
  for (int f = 0; f < 6; f++) bcgen = bcgen || (p.bc[f] != EMMA_RT_BC_PERIODIC);
  const bool diag = p.want_total != 0;
  cudaError_t e;
  switch (p.nst) {
    case 4: e = launch_nst<4>(p, maps_in, Uout, parts, nblk, diag, bcgen, st); break;
    case 8: e = launch_nst<8>(p, maps_in, Uout, parts, nblk, diag, bcgen, st); break;
    default: e = launch_nst<NST_DEFAULT>(p, maps_in, Uout, parts, nblk, diag, bcgen, st); break;
  }
  *n_parts = (diag || bcgen) ? nblk : 0;
  return e == cudaSuccess ? 1 : 0;
}

}  // namespace emma
