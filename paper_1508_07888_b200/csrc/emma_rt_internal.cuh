// emma_rt_internal.cuh -- shared declarations of the CUDA path (sm_100a).  Not part of the C-ABI.
//
// Internal storage differs from the C-ABI's units on purpose:
//   * radiation: float4 (N, phi_x, phi_y, phi_z) with phi = F / c_red  (same units as N; the whole
//     transport update then carries the single coefficient nu/2 = c_red dt / (2 dx));
//   * ionisation state: ONE float `xs` per cell: xs >= 0 means x = xs (x <= 1/2); xs < 0 means the NEUTRAL
//     fraction y = 1-x = -xs (x > 1/2).  Both ends keep full fp32 relative precision;
//   * energy: eps = e / n0  [erg per hydrogen atom], so T = eps / (1.5 k_B (1+x)).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/emma_rt.h"

namespace emma {

constexpr int MAXG = EMMA_RT_MAX_GROUPS;
constexpr int MAXL = EMMA_RT_MAX_LEVELS;
constexpr int MAX_PART_BLOCKS = 2048;          // max blocks of a chemistry kernel (each block writes one Partial)

// per-block partial diagnostics (fp64 sums in units of photons: already multiplied by the cell volume)
struct Partial {
  double total, injected, absorbed, recomb, outflow;
  float dtau_min;
  unsigned int nsub_max;
  unsigned long long nsub, nhalv, nonfinite, ndefer;
  unsigned int err;                            // bit 0: ESUBCYCLE
  unsigned int pad;
};

struct DiagDev {                               // device-resident, written by finalize_kernel
  emma_rt_diag d;
  unsigned int err_sticky;                     // OR of every step's flags since init (bit 0 ESUBCYCLE, bit 1 non-finite)
  unsigned int err_last;                       // flags of the last step
  unsigned int pad_bad;                        // host side only: invalid-input count read back by emma_rt_step_host
};

// physics + geometry constants of the chemistry kernels
struct ChemParams {
  int G, otsa, thermal, max_halvings, record;
  float dt;
  float csig[MAXG];        // c_red * sigma_N,g            [cm^3 s^-1]
  float csigE[MAXG];       // c_red * Sigma_E,g            [erg cm^3 s^-1]   Sigma_E = sigma_E <E> - sigma_N 13.6 eV
  float e_tol;
};

struct LevelDev {
  long long ncell;         // cells on this level
  long long nocts;         // octs (level >= 1)
  float* n0;
  float* xs;
  float* eps;
  unsigned int* subc;      // or nullptr
  int* parent;             // [nocts] split cell on the level below                     (level >= 1)
  int* anc0;               // [nocts] coarse ancestor cell                               (level >= 1)
  int* child;              // [ncell] oct on the level above or -1                       (1 <= level < n_levels)
  unsigned int* refined;   // bitmap over cells: split                                    (level 0 when n_levels > 0)
  float4* Ut;              // [G][nocts] restricted radiation of each oct, transient      (level >= 2)
  unsigned int* srcmask;   // bitmap over cells: hosts a source
  int* src_cell;           // [n_src] sorted cell ids
  float* src_S;            // [n_src][G] photons cm^-3 s^-1
  int n_src;
  double dV;               // cell volume [cm^3]
  double dV_total;         // = dV; 0 for a sweep that must not add to the photon total (see fold())
};

// Deferred octs of a refined level under CRTA (chemistry.cu: chem_refined_kernel and its tail)
struct CrtaQueue {
  int cap;                       // octs the side buffer holds
  int* oct_list;                 // [cap] slot -> oct of this level
  float4* side;                  // [G][cap * 8] radiation of the members of a deferred oct after the step
  int* lqueue;                   // [<= cap * 8] deferred leaves: slot * 8 + child
  unsigned int* counters;        // [0] leaves queued, [1] leaves taken by the tail, [2] octs deferred
};

struct TransportParams {
  int n, G;
  int bc[6];
  int zchunk, nzc, tiles_x, tiles_y;
  int z_lo, z_hi;          // planes [z_lo, z_hi) this launch covers (fused pass; the whole grid unless emma_rt_step_host slabs it)
  int nst;                 // stages of the TMA ring (transport_tma.cu)
  int pf;                  // planes ahead of the march that are prefetched into L2 (0 = off)
  int want_total;          // 1 when chemistry is off: the transport pass also sums N dV
  float nu;                // c_red dt / dx
  float c0, c1;            // 1 - 3 nu and nu / 2, rounded once from fp64
  float4 inflow[6][MAXG];  // ghost state (N, phi) of EMMA_RT_BC_INFLOW faces, per group (reading A20)
  double dV;
};

// TMA descriptors of one radiation buffer (transport_tma.cu): the tile's own 32 x 16 box, a 32 x 1 halo row, a
// 1 x 16 halo column
struct TransportMaps {
  CUtensorMap main, row, col;
};

// Optional per-kernel device timing: CUDA events recorded on the handle's stream around every launch of a step.
struct Profiler {
  struct Span { int kind; cudaEvent_t a, b; };
  bool on = false;
  cudaStream_t st = 0;
  std::vector<cudaEvent_t> pool;
  size_t used = 0;
  std::vector<Span> spans;
  cudaEvent_t get()
  {
    if (used == pool.size()) { cudaEvent_t e; cudaEventCreate(&e); pool.push_back(e); }
    return pool[used++];
  }
  void begin(int kind)
  {
    if (!on) return;
    Span s{kind, get(), get()};
    cudaEventRecord(s.a, st);
    spans.push_back(s);
  }
  void end()
  {
    if (on) cudaEventRecord(spans.back().b, st);
  }
  void reset() { spans.clear(); used = 0; }
};

// ---- launchers (each returns the number of kernels it launched) ---------------------------------------------
int launch_transport(const TransportParams& p, const float4* Uin, float4* Uout, Partial* parts, int* n_parts,
                     cudaStream_t st);
int make_transport_maps(const float4* U, int n, int G, TransportMaps* out, int tile_y = 16, int tile_x = 32, int main_x = 0);
int launch_transport_tma(const TransportParams& p, const TransportMaps& maps_in, float4* Uout, Partial* parts,
                         int* n_parts, cudaStream_t st);
int launch_chem_level0(const ChemParams& cp, const LevelDev& L0, float4* U, long long ncell, int* queue,
                       unsigned int* qcount, Partial* parts, int* n_parts, int sm_count, int ctas_per_sm, cudaStream_t st,
                       Profiler* pf);
// per-device set-up of the kernels that need more than 48 KB of dynamic shared memory; called by emma_rt_init for every
// handle with the handle's device current (function attributes belong to the device's context, not to the process)
cudaError_t configure_transport_tma();
cudaError_t configure_transport_hll();
cudaError_t configure_fused(int G);
cudaError_t configure_chemistry(int G, int* ctas_per_sm);
int launch_chem_tail(const ChemParams& cp, const LevelDev& L0, float4* U, long long ncell, int* queue,
                     unsigned int* qcount, Partial* parts, int* n_parts, int sm_count, cudaStream_t st, Profiler* pf);
int launch_fused(const TransportParams& p, const TransportMaps& maps_in, float4* Uout, const ChemParams& cp,
                 const LevelDev& L0, int* queue, unsigned int* qcount, Partial* parts, int* n_parts, cudaStream_t st);
int fused_ctas_per_sm();
int fused_tile_y();
int launch_transport_hll(const TransportParams& p, const TransportMaps& maps_in, float4* Uout, Partial* parts,
                         int* n_parts, cudaStream_t st);
int hll_ctas_per_sm();
int hll_tile_x();
int hll_main_x();
int launch_chem_refined(const ChemParams& cp, const LevelDev* lv, int level, int n_levels, float4* U,
                        long long ncell0, const CrtaQueue& q, Partial* parts, int* n_parts, int sm_count, cudaStream_t st);
int launch_inject_sources(const LevelDev& L0, int G, float dt, float4* U, long long ncell0, Partial* parts,
                          int* n_parts, cudaStream_t st);
int launch_finalize(const Partial* parts, int n_parts, DiagDev* diag, unsigned int* qcount, double t_sim,
                    cudaStream_t st);
int launch_restrict_init(const LevelDev* lv, int level, cudaStream_t st);
// conversions between the C-ABI's units and the internal storage (one chunk of cells)
int launch_export(int field, const LevelDev& L, const float4* Ug, float c_red, long long off, long long cnt,
                  void* dst, cudaStream_t st);
int launch_import(int field, const LevelDev& L, float4* Ug, float c_red, long long off, long long cnt,
                  const void* src, unsigned int* bad, cudaStream_t st);
// sum of n float4.x values times dV -> *out (fp64, fixed summation order); scratch = >= 1024 Partial slots
int launch_sum_N(const float4* U, long long n, double dV, Partial* scratch, double* out, cudaStream_t st);
int launch_set_bits(unsigned int* mask, const int* cells, int n, cudaStream_t st);

// ---- small device helpers -----------------------------------------------------------------------------------
__device__ __forceinline__ float frcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float fsqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float fex2(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float flg2(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ unsigned long long warp_sum(unsigned long long v)
{
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// per-thread accumulators -> one Partial per block (fixed-shape tree: xor-shuffle inside a warp, then warps in
// index order), so a launch's partials do not depend on scheduling
struct Acc {
  double total = 0, injected = 0, absorbed = 0, recomb = 0, outflow = 0;
  float dtau_min = __builtin_huge_valf();
  unsigned int nsub_max = 0, err = 0;
  unsigned long long nsub = 0, nhalv = 0, nonfinite = 0, ndefer = 0;
};

__device__ inline void block_reduce_store(const Acc& a, Partial* out)
{
  __shared__ Partial s_part[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
  Partial p;
  p.total = warp_sum(a.total); p.injected = warp_sum(a.injected); p.absorbed = warp_sum(a.absorbed);
  p.recomb = warp_sum(a.recomb); p.outflow = warp_sum(a.outflow);
  float m = a.dtau_min;
  unsigned int mx = a.nsub_max, er = a.err;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    m = fminf(m, __shfl_xor_sync(0xffffffffu, m, o));
    mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    er |= __shfl_xor_sync(0xffffffffu, er, o);
  }
  p.dtau_min = m; p.nsub_max = mx; p.err = er; p.pad = 0;
  p.nsub = warp_sum(a.nsub); p.nhalv = warp_sum(a.nhalv); p.nonfinite = warp_sum(a.nonfinite);
  p.ndefer = warp_sum(a.ndefer);
  if (lane == 0) s_part[warp] = p;
  __syncthreads();
  if (threadIdx.x == 0) {
    Partial t = s_part[0];
    for (int w = 1; w < nwarp; w++) {
      const Partial& q = s_part[w];
      t.total += q.total; t.injected += q.injected; t.absorbed += q.absorbed; t.recomb += q.recomb;
      t.outflow += q.outflow; t.dtau_min = fminf(t.dtau_min, q.dtau_min); t.nsub_max = max(t.nsub_max, q.nsub_max);
      t.err |= q.err; t.nsub += q.nsub; t.nhalv += q.nhalv; t.nonfinite += q.nonfinite; t.ndefer += q.ndefer;
    }
    *out = t;
  }
}

}  // namespace emma

// ---- standard (non-CRTA) AMR transport, reading A21 (amr.cu) -------------------------------------------
namespace emma {

// device view of the level hierarchy in AMR-transport mode.  Every level carries its own radiation; `nbr` is the
// paper's oct structure ("6 pointers toward the 6 Cartesian neighbors cells of c^{l-1}").
struct AmrDev {
  int nl, n, G;
  int bc[6];
  long long ncell[MAXL + 1];
  float4* U[MAXL + 1];          // current radiation of the level, [G][ncell]
  float4* dU[MAXL + 1];         // [G][ucap] change of a fine cell by its face towards a coarser leaf, one record per face of the
                                // host-built list (levels >= 1)
  float4* depS[MAXL + 1];       // [G][scap] what an oct side hands to the coarse leaf behind it over the level's two sub-steps of the
                                // coarse step (Fig. 3 (i)-(ii)), one record per (oct, face) (levels >= 1)
  long long ucap[MAXL + 1], scap[MAXL + 1];
  const int* child[MAXL + 1];   // [ncell] oct on the level above or -1 (levels < nl)
  const int* nbr[MAXL + 1];     // [nocts][6] cell of the level below next to the oct's parent cell in -x,+x,-y,+y,-z,+z,
                                // or -1 - bc for a non-periodic box face (levels >= 1)
  const int* nbo[MAXL + 1];     // [nocts][6] derived for the static mesh: the oct of the SAME level behind each face of the
                                // oct; -16 - s if that side is a coarser leaf (s = the side's record index); -2 - bc for a
                                // non-periodic box face (levels >= 1)
  const unsigned int* hasdep[MAXL + 1];   // bitmap over the cells of a level: a leaf with a split face neighbour of its own
                                          // level, i.e. one that receives deposits (1 <= level < nl)
  float4 inflow[6][MAXG];
};

int launch_amr_transport(const AmrDev& A, int level, float nuh, float4* Unew, double dV, int hll, Partial* parts, int* n_parts,
                         cudaStream_t st);
int launch_amr_ghost_faces(const AmrDev& A, int level, float nuh, int sub, const int* slot_cell, const int* slot_coarse,
                           const unsigned char* slot_face, const int* slot_refs, int n_slots, int hll, cudaStream_t st);
int launch_amr_chem(const ChemParams& cp, const LevelDev& L, const AmrDev& A, int level, int count_total, int limit,
                    Partial* parts, int* n_parts, cudaStream_t st);
int launch_amr_sources(const LevelDev& L, const AmrDev& A, int level, float dt, int count_total, int limit, Partial* parts,
                       int* n_parts, cudaStream_t st);
int launch_amr_restrict(const LevelDev& Lfine, const LevelDev& Lcoarse, const AmrDev& A, int level_fine, int with_gas,
                        cudaStream_t st);
int launch_amr_inject_init(const LevelDev& Lfine, const AmrDev& A, int level_fine, cudaStream_t st);
int launch_amr_fix0(const AmrDev& A, const float4* Uold, float4* Unew, const int* fix_cell, const unsigned char* fix_mask,
                    int n_fix, float nuh, int hll, cudaStream_t st);
int launch_amr_outflow0(const AmrDev& A, const float4* Uold, float nuh, double dV, int hll, Partial* parts, int* n_parts,
                        cudaStream_t st);

}  // namespace emma
