// api.cu -- host side of the C-ABI (include/emma_rt.h): validation, arena layout, AMR index arrays, sources,
// the step loop (kernel sequence of SURVEY.md section 3(c)) and field I/O.  No compute happens on the host; without
// a CUDA device every entry point that needs one fails with EMMA_RT_ECUDA.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <unordered_map>
#include <vector>

#include "emma_rt_internal.cuh"

using namespace emma;

namespace {

constexpr size_t ALIGN = 256;
constexpr int PART_SLOTS = 106496;       // worst case of a 3-level standard-AMR step: 15 level sweeps x 3 grids of <= MAX_PART_BLOCKS
                                         // (transport, chemistry main, tail) + one dense transport grid (9.4 MB)
constexpr int TRANSPORT_MAX_BLOCKS = 8192;
constexpr double E_HI_ERG = 13.6 * 1.602176634e-12;          // "E_13.6" of PAPER.md:266

size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

struct Layout {
  size_t U[2];
  size_t n0[MAXL + 1], xs[MAXL + 1], eps[MAXL + 1], subc[MAXL + 1];
  size_t refined0;
  size_t parent[MAXL + 1], anc0[MAXL + 1], child[MAXL + 1], Ut[MAXL + 1];
  size_t srcmask[MAXL + 1], src_cell[MAXL + 1], src_S[MAXL + 1];
  size_t queue, qcount, parts, diag;
  size_t host_stage;                                // one exported slab of emma_rt_step_host: U (G float4) + x + T
  size_t crta_oct[MAXL + 1], crta_side[MAXL + 1];   // deferred octs of the refined levels under CRTA (chemistry.cu)
  // standard AMR transport (A21): per-level radiation (double-buffered), deposits, oct neighbour pointers, level-0
  // child index and the list of level-0 leaves that touch a split cell
  size_t aU[2][MAXL + 1], adU[MAXL + 1], adepS[MAXL + 1], anbr[MAXL + 1], anbo[MAXL + 1], achild0, afix_cell, afix_mask;
  size_t aslot_cell[MAXL + 1], aslot_coarse[MAXL + 1], aslot_face[MAXL + 1], aslot_refs[MAXL + 1], ahasdep[MAXL + 1], arefined[MAXL + 1];   // faces of refined leaves towards a coarser leaf
  size_t total;
};

struct Shape {
  int n, G, nl;
  long long ncell[MAXL + 1], nocts[MAXL + 1];
  long long max_src;
  bool record, need_queue, amr;
  long long crta_cap[MAXL + 1];
  int slab_planes;                              // planes per slab of emma_rt_step_host (0: not available)                 // octs the side buffer of a refined level holds (0: none)
};

bool make_shape(const emma_rt_config* c, const emma_rt_amr* a, Shape& s)
{
  if (!c || c->struct_size != sizeof(emma_rt_config) || c->abi_version != EMMA_RT_ABI_VERSION) return false;
  if (c->n_coarse < 2 || c->n_coarse > 1290 || c->n_groups < 1 || c->n_groups > MAXG) return false;
  for (int f = 0; f < 6; f++)
    if (c->bc[f] < 0 || c->bc[f] > EMMA_RT_BC_INFLOW) return false;
  for (int d = 0; d < 3; d++)                                   // periodic faces come in pairs
    if ((c->bc[2 * d] == EMMA_RT_BC_PERIODIC) != (c->bc[2 * d + 1] == EMMA_RT_BC_PERIODIC)) return false;
  if (!(c->box_len_cm > 0) || !(c->c_red_cm_s > 0) || !(c->e_tol > 0) || c->max_halvings < 0) return false;
  for (int g = 0; g < c->n_groups; g++)
    if (!(c->sigma_N[g] >= 0) || !(c->sigma_E[g] >= 0) || !(c->E_mean[g] >= 0)) return false;
  s.n = c->n_coarse; s.G = c->n_groups;
  s.nl = a ? a->n_levels : 0;
  if (s.nl < 0 || s.nl > MAXL) return false;
  s.ncell[0] = (long long)s.n * s.n * s.n; s.nocts[0] = 0;
  if (s.nl > 0 && (!a->n_octs || !a->parent)) return false;
  for (int l = 1; l <= s.nl; l++) {
    if (a->n_octs[l - 1] > 0 && !a->parent[l - 1]) return false;
    if (a->n_octs[l - 1] < 0 || a->n_octs[l - 1] > s.ncell[l - 1] || 8 * a->n_octs[l - 1] > 2000000000LL)
      return false;
    s.nocts[l] = a->n_octs[l - 1];
    s.ncell[l] = 8 * s.nocts[l];
  }
  s.max_src = c->max_source_cells > 0 ? c->max_source_cells : 65536;
  s.record = c->record_subcycles != 0;
  s.need_queue = c->chemistry != 0 && c->thermal != 0;
  if (c->amr_transport != 0 && c->amr_transport != 1) return false;
  s.amr = c->amr_transport == 1 && s.nl > 0;
  // emma_rt_step_host streams the state through the device in z-slabs: ~32 slabs, at least 8 planes each
  s.slab_planes = (s.nl == 0 && c->chemistry != 0) ? std::min(s.n, std::max(8, s.n / 32)) : 0;
  for (int l = 0; l <= MAXL; l++) s.crta_cap[l] = 0;
  if (!s.amr && s.need_queue)                   // a side-buffer slot for every oct: any number of octs can be deferred
    for (int l = 1; l <= s.nl; l++) s.crta_cap[l] = s.nocts[l];
  if (s.amr && s.nl > 3) return false;          // partial-sum slots: 2^(nl+1) - 1 level sweeps per step
  return true;
}

void make_layout(const Shape& s, Layout& L)
{
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + (bytes ? bytes : 1)); return o; };
  memset(&L, 0, sizeof L);
  for (int b = 0; b < 2; b++) L.U[b] = take((size_t)s.G * s.ncell[0] * sizeof(float4));
  for (int l = 0; l <= s.nl; l++) {
    L.n0[l] = take(s.ncell[l] * 4); L.xs[l] = take(s.ncell[l] * 4); L.eps[l] = take(s.ncell[l] * 4);
    L.subc[l] = s.record ? take(s.ncell[l] * 4) : 0;
    const size_t words = (size_t)(s.ncell[l] + 31) / 32;
    L.srcmask[l] = take(words * 4);
    L.src_cell[l] = take(s.max_src * 4);
    L.src_S[l] = take(s.max_src * s.G * 4);
    if (l >= 1) {
      L.parent[l] = take(s.nocts[l] * 4);
      L.anc0[l] = take(s.nocts[l] * 4);
      if (l < s.nl) L.child[l] = take(s.ncell[l] * 4);
      if (l >= 2) L.Ut[l] = take((size_t)s.G * s.nocts[l] * sizeof(float4));
    }
  }
  L.refined0 = s.nl > 0 ? take((size_t)(s.ncell[0] + 31) / 32 * 4) : 0;
  long long qcells = s.ncell[0];
  if (s.amr) for (int l = 1; l <= s.nl; l++) qcells = std::max(qcells, s.ncell[l]);   // every level runs the two-pass chemistry
  for (int l = 1; l <= s.nl; l++) qcells = std::max(qcells, 8 * s.crta_cap[l]);
  L.queue = s.need_queue ? take(qcells * 4) : 0;
  L.qcount = take(256);
  for (int l = 1; l <= s.nl; l++)
    if (s.crta_cap[l] > 0) {
      L.crta_oct[l] = take((size_t)s.crta_cap[l] * 4);
      L.crta_side[l] = take((size_t)s.G * s.crta_cap[l] * 8 * sizeof(float4));
    }
  L.host_stage = s.slab_planes ? take((size_t)s.slab_planes * s.n * s.n * (16 * (size_t)s.G + 8)) : 0;
  L.parts = take((size_t)PART_SLOTS * sizeof(Partial));
  L.diag = take(sizeof(DiagDev));
  if (s.amr) {
    for (int l = 0; l <= s.nl; l++) {
      if (l >= 1) {
        for (int b = 0; b < 2; b++) L.aU[b][l] = take((size_t)s.G * s.ncell[l] * sizeof(float4));
        L.anbr[l] = take((size_t)s.nocts[l] * 6 * 4);
        L.anbo[l] = take((size_t)s.nocts[l] * 6 * 4);
        // capacity: every face cell of every oct (24 per oct); the list built at init is normally a small fraction
        L.aslot_cell[l] = take((size_t)s.nocts[l] * 24 * 4);
        L.aslot_coarse[l] = take((size_t)s.nocts[l] * 24 * 4);
        L.aslot_face[l] = take((size_t)s.nocts[l] * 24);
        L.aslot_refs[l] = take((size_t)s.nocts[l] * 6 * 6 * 4);     // 6 neighbour references per oct side
        // what a coarse-facing face does to its fine cell (one record per face and group) and what an oct side hands to
        // its coarse leaf (one record per side and group, summed over the two sub-steps): written by amr_ghost_faces_kernel, read by the cell
        // kernels of the two levels -- no read-modify-write, no atomics.  Worst-case capacity, like the lists
        L.adU[l] = take((size_t)s.G * s.nocts[l] * 24 * sizeof(float4));
        L.adepS[l] = take((size_t)s.G * s.nocts[l] * 6 * sizeof(float4));
        L.ahasdep[l] = take((size_t)(s.ncell[l] + 31) / 32 * 4);
        L.arefined[l] = take((size_t)(s.ncell[l] + 31) / 32 * 4);     // split cells of the level (chemistry skips them)
      }
    }
    L.achild0 = take((size_t)s.ncell[0] * 4);
    L.afix_cell = take((size_t)s.nocts[1] * 6 * 4);
    L.afix_mask = take((size_t)s.nocts[1] * 6);
  }
  L.total = off;
}

// Tuning knobs for experiments, read ONCE from the environment by emma_rt_init (documented in include/emma_rt.h) and
// clamped to their valid ranges; 0 / unset = the built-in choice.
struct Tune {
  int nzc = 0;          // EMMA_RT_TUNE_NZC      z-chunks per tile column of the dense passes (0: cost model)
  int nst = 6;          // EMMA_RT_TUNE_NST      stages of the TMA ring of transport_tma_kernel: 4, 6 or 8
  int tma = 1;          // EMMA_RT_TUNE_TMA      0: the non-TMA transport kernel (transport.cu)
  int fused = 1;        // EMMA_RT_TUNE_FUSED    0: two-pass schedule whatever emma_rt_set_schedule says
  int chem_ctas = 0;    // EMMA_RT_TUNE_CHEMCTAS persistent CTAs per SM of the chemistry main pass (0: occupancy)
};

int env_int(const char* name, int dflt, int lo, int hi)
{
  const char* v = getenv(name);
  if (!v || !*v) return dflt;
  char* end = nullptr;
  const long x = strtol(v, &end, 10);
  if (end == v || x < lo || x > hi) return dflt;     // out of range or not a number: ignored
  return (int)x;
}

}  // namespace

struct emma_rt {
  emma_rt_config cfg;
  Tune tune;
  int chem_ctas_per_sm;                        // CTAs of the chemistry main pass that fit on an SM of this device
  Shape sh;
  Layout lay;
  char* arena;
  cudaStream_t st;
  int sm_count;
  int cur;                                     // U[cur] holds the current radiation field
  LevelDev lv[MAXL + 1];
  std::unordered_map<long long, int> child_of[MAXL + 1];   // split cell -> oct on the level above (host copy)
  std::vector<int> anc0_h[MAXL + 1];
  double dx, t_sim;
  long long launches;
  DiagDev* diag_pinned;
  Profiler prof;
  TransportMaps tmaps[2];                      // TMA descriptors of U[0], U[1]
  TransportMaps tmaps_f[2];                    // the same with the fused pass's tile height
  TransportMaps tmaps_h[2];                    // the same with the HLL pass's tile width
  int fused;                                   // schedule of the coupled step (emma_rt_set_schedule)
  int flux;                                    // interface flux of the transport update (emma_rt_set_flux)
  float4 inflow[6][MAXG];                      // ghost state (N, phi) of inflow faces (emma_rt_set_inflow)
  // standard AMR transport (A21)
  int acur[MAXL + 1];                          // aU[acur[l]][l] holds the current radiation of refined level l
  int n_fix;                                   // level-0 leaves with a split face neighbour
  int n_slots[MAXL + 1];                       // faces of the leaves of a refined level towards a coarser leaf
  bool amr_dirty;                              // U was written: restrict bottom-up before the next step
  cudaStream_t s_in = nullptr, s_out = nullptr;  // copy streams of emma_rt_step_host (created at its first call)
  std::vector<cudaEvent_t> ev_in, ev_c;          // per slab: inputs on the device / slab computed
  cudaEvent_t ev_start = nullptr;
  char err[256];

  float4* U(int b) const { return (float4*)(arena + lay.U[b]); }
  float4* Ulev(int l, int other = 0) const       // current (other = 0) or scratch radiation buffer of a level
  {
    if (l == 0) return U(other ? 1 - cur : cur);
    return (float4*)(arena + lay.aU[other ? 1 - acur[l] : acur[l]][l]);
  }
  Partial* parts() const { return (Partial*)(arena + lay.parts); }
  CrtaQueue crta_queue(int l) const
  {
    CrtaQueue q;
    q.cap = (int)sh.crta_cap[l];
    q.oct_list = q.cap ? (int*)(arena + lay.crta_oct[l]) : nullptr;
    q.side = q.cap ? (float4*)(arena + lay.crta_side[l]) : nullptr;
    q.lqueue = q.cap ? (int*)(arena + lay.queue) : nullptr;
    q.counters = (unsigned int*)(arena + lay.qcount);
    return q;
  }
  unsigned int* qcount() const { return (unsigned int*)(arena + lay.qcount); }
  DiagDev* diag() const { return (DiagDev*)(arena + lay.diag); }
};

namespace {

int fail(emma_rt* h, int code, const char* fmt, ...)
{
  if (h) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(h->err, sizeof h->err, fmt, ap);
    va_end(ap);
  }
  return code;
}

// Every entry point that launches work runs through here: the handle's device is made current (a process may hold
// handles on several GPUs) and nothing thrown by the host-side bookkeeping (std::bad_alloc of its vectors and maps)
// crosses the C boundary.
template <class F>
int guarded(emma_rt* h, bool set_device, F&& f)
{
  try {
    if (h && set_device) {
      const cudaError_t e = cudaSetDevice(h->cfg.device);
      if (e != cudaSuccess) return fail(h, EMMA_RT_ECUDA, "cudaSetDevice(%d): %s", h->cfg.device, cudaGetErrorString(e));
    }
    return f();
  } catch (const std::bad_alloc&) {
    return fail(h, EMMA_RT_ENOMEM, "out of host memory");
  } catch (...) {
    return fail(h, EMMA_RT_EINVAL, "internal error (exception)");
  }
}

#define CUDA_TRY(h, call)                                                                       \
  do {                                                                                          \
    cudaError_t e__ = (call);                                                                   \
    if (e__ != cudaSuccess) return fail(h, EMMA_RT_ECUDA, "%s: %s", #call, cudaGetErrorString(e__)); \
  } while (0)

// chem_level0 opens its own profiler spans; inside an AMR sweep the outer AMR_CHEM span already covers it
Profiler* nullptr_prof(emma_rt* h)
{
  static thread_local Profiler off;            // on = false: begin/end do nothing
  (void)h;
  return &off;
}

// device view of the hierarchy in AMR-transport mode, with the buffers that are current right now
AmrDev amr_view(const emma_rt* h)
{
  AmrDev A;
  memset(&A, 0, sizeof A);
  const Shape& s = h->sh;
  A.nl = s.nl; A.n = s.n; A.G = s.G;
  for (int f = 0; f < 6; f++) A.bc[f] = h->cfg.bc[f];
  memcpy(A.inflow, h->inflow, sizeof A.inflow);
  for (int l = 0; l <= s.nl; l++) {
    A.ncell[l] = s.ncell[l];
    A.U[l] = h->Ulev(l);
    A.dU[l] = l >= 1 ? (float4*)(h->arena + h->lay.adU[l]) : nullptr;
    A.depS[l] = l >= 1 ? (float4*)(h->arena + h->lay.adepS[l]) : nullptr;
    A.ucap[l] = 24 * s.nocts[l]; A.scap[l] = 6 * s.nocts[l];
    A.child[l] = l == 0 ? (const int*)(h->arena + h->lay.achild0) : l < s.nl ? h->lv[l].child : nullptr;
    A.nbr[l] = l >= 1 ? (const int*)(h->arena + h->lay.anbr[l]) : nullptr;
    A.nbo[l] = l >= 1 ? (const int*)(h->arena + h->lay.anbo[l]) : nullptr;
    A.hasdep[l] = (l >= 1 && l < s.nl) ? (const unsigned int*)(h->arena + h->lay.ahasdep[l]) : nullptr;
  }
  return A;
}

// One emma_rt_step call in AMR-transport mode (reading A21): the recursion advance(l, dt) = advance(l+1, dt/2) x 2
// -> transport(l) -> chemistry(l) -> restrict(l+1 -> l), flattened into a list of level sweeps per coarse step.
int step_amr(emma_rt* h, double dt, int n_steps, TransportParams& tp, const TransportParams& hp, const ChemParams& cp,
             bool use_tma, bool hll)
{
  const Shape& s = h->sh;
  const double c = h->cfg.c_red_cm_s;
  // standard AMR scheme (A21): advance(l, dt) = advance(l+1, dt/2) x 2 -> transport(l) -> chemistry(l) -> restrict(l+1 -> l)
  const int ihll = hll ? 1 : 0;
  const float nuh = (float)(0.5 * (c * dt / h->dx));           // the same CFL number on every level
  tp.want_total = 0;
  bool open_faces = false;
  for (int f = 0; f < 6; f++) open_faces = open_faces || h->cfg.bc[f] != EMMA_RT_BC_PERIODIC;
  if (h->amr_dirty) {                                          // U was written: split cells := children mean
    for (int l = s.nl; l >= 1; l--) h->launches += launch_amr_restrict(h->lv[l], h->lv[l - 1], amr_view(h), l, 0, h->st);
    h->amr_dirty = false;
  }
  // (level, dt, last sub-step of the level in this coarse step) in execution order, finest first
  struct Call { int l; double dt; bool last; };
  std::vector<Call> order;
  struct Rec { static void go(std::vector<Call>& o, int l, int nl, const long long* nc, double dtl, bool last) {
    if (l < nl && nc[l + 1] > 0) { go(o, l + 1, nl, nc, 0.5 * dtl, false); go(o, l + 1, nl, nc, 0.5 * dtl, last); }
    o.push_back({l, dtl, last});
  } };
  Rec::go(order, 0, s.nl, s.ncell, dt, true);
  int sub_of[MAXL + 1] = {0};                     // a refined level is swept twice per step of the level below: first / second sub-step
  // worst-case partial-sum slots of one coarse step, checked BEFORE the first launch so that a refusal leaves the state
  // untouched: every sweep may use a transport grid, a chemistry main grid and a tail grid
  if ((long long)order.size() * 3 * MAX_PART_BLOCKS + TRANSPORT_MAX_BLOCKS > PART_SLOTS)
    return fail(h, EMMA_RT_EINVAL, "too many level sweeps for the partial-sum slots");
  for (int step = 0; step < n_steps; step++) {
    int off = 0;
    Partial* P = h->parts();
    for (const Call& cl : order) {
      const int l = cl.l;
      int np = 0;
      if (l == 0) {
        // dense pass over the whole block (its partials are not used: split cells must not count), then the
        // sparse correction of the leaves that touch a split cell
        h->prof.begin(EMMA_RT_K_TRANSPORT);
        if (hll) {
          const int k = launch_transport_hll(hp, h->tmaps_h[h->cur], h->U(1 - h->cur), P + off, &np, h->st);
          if (!k) return fail(h, EMMA_RT_ECUDA, "HLL transport launch failed: %s", cudaGetErrorString(cudaGetLastError()));
          h->launches += k;
        } else if (use_tma) {
          const int k = launch_transport_tma(tp, h->tmaps[h->cur], h->U(1 - h->cur), P + off, &np, h->st);
          if (!k) return fail(h, EMMA_RT_ECUDA, "transport launch failed: %s", cudaGetErrorString(cudaGetLastError()));
          h->launches += k;
        } else h->launches += launch_transport(tp, h->U(h->cur), h->U(1 - h->cur), P + off, &np, h->st);
        h->prof.end();
        AmrDev A = amr_view(h);
        h->prof.begin(EMMA_RT_K_OTHER);
        if (open_faces) { h->launches += launch_amr_outflow0(A, h->U(h->cur), nuh, h->lv[0].dV, ihll, P + off, &np, h->st); off += np; }
        h->launches += launch_amr_fix0(A, h->U(h->cur), h->U(1 - h->cur), (const int*)(h->arena + h->lay.afix_cell),
                                       (const unsigned char*)(h->arena + h->lay.afix_mask), h->n_fix, nuh, ihll, h->st);
        h->prof.end();
        h->cur = 1 - h->cur;
        if (h->cfg.chemistry) {
          h->launches += launch_chem_level0(cp, h->lv[0], h->U(h->cur), s.ncell[0], (int*)(h->arena + h->lay.queue), h->qcount(),
                                            P + off, &np, h->sm_count, h->chem_ctas_per_sm, h->st, &h->prof);
          off += np;
        } else {
          h->prof.begin(EMMA_RT_K_OTHER);
          h->launches += launch_amr_sources(h->lv[0], amr_view(h), 0, (float)dt, 1, 0, P + off, &np, h->st);
          h->prof.end();
          off += np;
        }
      } else {
        AmrDev A = amr_view(h);
        h->prof.begin(EMMA_RT_K_AMR_TRANSPORT);
        // the faces towards a coarser leaf first: from the start-of-step states they write the per-face change records the
        // cell kernel adds to its result and the per-side records the coarse leaf gathers when ITS step comes
        h->launches += launch_amr_ghost_faces(A, l, nuh, sub_of[l], (const int*)(h->arena + h->lay.aslot_cell[l]),
                                              (const int*)(h->arena + h->lay.aslot_coarse[l]),
                                              (const unsigned char*)(h->arena + h->lay.aslot_face[l]),
                                              (const int*)(h->arena + h->lay.aslot_refs[l]), h->n_slots[l], ihll, h->st);
        sub_of[l] ^= 1;
        h->launches += launch_amr_transport(A, l, nuh, h->Ulev(l, 1), h->lv[l].dV, ihll, P + off, &np, h->st);
        h->prof.end();
        off += np;
        h->acur[l] = 1 - h->acur[l];
        A = amr_view(h);
        ChemParams cl_cp = cp;
        cl_cp.dt = (float)cl.dt;
        h->prof.begin(EMMA_RT_K_AMR_CHEM);
        if (h->cfg.chemistry && !hll) {
          // the two-pass chemistry of level 0 (bulk-async main pass + compacted tail, chemistry.cu) on this level's arrays
          LevelDev Lc = h->lv[l];
          Lc.refined = l < s.nl ? (unsigned int*)(h->arena + h->lay.arefined[l]) : nullptr;
          Lc.dV_total = cl.last ? Lc.dV : 0.0;
          h->launches += launch_chem_level0(cl_cp, Lc, h->Ulev(l), s.ncell[l], (int*)(h->arena + h->lay.queue), h->qcount(),
                                            P + off, &np, h->sm_count, h->chem_ctas_per_sm, h->st, nullptr_prof(h));
          CUDA_TRY(h, cudaMemsetAsync(h->qcount(), 0, 8, h->st));      // queue counters of the next sweep
        } else if (h->cfg.chemistry) h->launches += launch_amr_chem(cl_cp, h->lv[l], A, l, cl.last ? 1 : 0, ihll, P + off, &np, h->st);
        else h->launches += launch_amr_sources(h->lv[l], A, l, (float)cl.dt, cl.last ? 1 : 0, ihll, P + off, &np, h->st);
        h->prof.end();
        off += np;
      }
      if (l < s.nl && s.ncell[l + 1] > 0) {
        h->prof.begin(EMMA_RT_K_OTHER);
        h->launches += launch_amr_restrict(h->lv[l + 1], h->lv[l], amr_view(h), l + 1, h->cfg.chemistry ? 1 : 0, h->st);
        h->prof.end();
      }
    }
    h->t_sim += dt;
    h->prof.begin(EMMA_RT_K_FINALIZE);
    h->launches += launch_finalize(P, off, h->diag(), h->qcount(), h->t_sim, h->st);
    h->prof.end();
  }
  return EMMA_RT_OK;
}

// Index arrays of the AMR-transport mode (reading A21, section 4), built once on the host for the static mesh:
// the paper's oct neighbour pointers (the 6 cells of level l-1 around the oct's parent cell) and what the
// kernels read, derived from them: same-level neighbour octs, the level-0 child index, the receivers of deposits, the
// faces towards a coarser leaf with their six resolved coarse references, the level-0 leaves that touch a split cell.
// A face jump > 1 is refused here.
int init_amr_topology(emma_rt* h, const std::vector<std::vector<int>>& parent_h, const std::vector<std::vector<int>>& child_h)
{
  const Shape& s = h->sh;
  std::vector<std::vector<int>> nbr_h(s.nl + 1);
  std::vector<int> child0_h, fix_cell_h;
  std::vector<unsigned char> fix_mask_h;
  std::vector<std::vector<int>> slot_cell_h(s.nl + 1), slot_coarse_h(s.nl + 1), nbo_h(s.nl + 1), slot_refs_h(s.nl + 1);
  std::vector<std::vector<unsigned char>> slot_face_h(s.nl + 1);
  std::vector<std::vector<unsigned int>> hasdep_h(s.nl + 1), refined_lv_h(s.nl + 1);
  const int n = s.n;
  auto bc_code = [&](int a, int side) { return -1 - h->cfg.bc[2 * a + side]; };       // non-periodic box face
  // neighbour of a level-0 cell, or the box-face code
  auto nb0 = [&](long long cell, int a, int side) -> long long {
    const long long stride = a == 0 ? 1 : a == 1 ? n : (long long)n * n;
    const int ca = a == 0 ? (int)(cell % n) : a == 1 ? (int)((cell / n) % n) : (int)(cell / ((long long)n * n));
    const int cn = ca + (side ? 1 : -1);
    if (cn < 0 || cn >= n) {
      if (h->cfg.bc[2 * a + side] != EMMA_RT_BC_PERIODIC) return bc_code(a, side);
      return cell + (side ? -(long long)(n - 1) : (long long)(n - 1)) * stride;
    }
    return cell + (side ? stride : -stride);
  };
  for (int l = 1; l <= s.nl; l++) {
    nbr_h[l].resize((size_t)s.nocts[l] * 6);
    for (long long o = 0; o < s.nocts[l]; o++) {
      const long long p = parent_h[l][o];                      // the oct's parent cell, on level l-1
      for (int a = 0; a < 3; a++)
        for (int side = 0; side < 2; side++) {
          long long q;
          if (l == 1) q = nb0(p, a, side);
          else {
            const long long po = p >> 3;                       // the parent cell's own oct (level l-1)
            const int k = (int)(p & 7), bit = (k >> a) & 1;
            if (side != bit) q = (po << 3) | (k ^ (1 << a));
            else {
              const int pp = nbr_h[l - 1][po * 6 + 2 * a + side];     // cell of level l-2
              if (pp < 0) q = pp;
              else {
                auto it = h->child_of[l - 2].find(pp);
                if (it == h->child_of[l - 2].end())
                  return fail(h, EMMA_RT_EINVAL, "resolution jump > 1 across a face of oct %lld of level %d (PAPER.md:75)", o, l);
                q = ((long long)it->second << 3) | (k ^ (1 << a));
              }
            }
          }
          nbr_h[l][o * 6 + 2 * a + side] = (int)q;
        }
    }
    CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.anbr[l], nbr_h[l].data(), nbr_h[l].size() * 4, cudaMemcpyHostToDevice, h->st));
  }
  child0_h.assign((size_t)s.ncell[0], -1);
  for (auto& kv : h->child_of[0]) child0_h[kv.first] = kv.second;
  CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.achild0, child0_h.data(), child0_h.size() * 4, cudaMemcpyHostToDevice, h->st));
  // same-level neighbour octs, derived from the neighbour-cell pointers
  for (int l = 1; l <= s.nl; l++) {
    nbo_h[l].resize((size_t)s.nocts[l] * 6);
    for (size_t i = 0; i < nbo_h[l].size(); i++) {
      const int pcell = nbr_h[l][i];
      if (pcell < 0) { nbo_h[l][i] = pcell - 1; continue; }              // -1 - bc  ->  -2 - bc
      nbo_h[l][i] = (l == 1) ? child0_h[pcell] : child_h[l - 1][pcell];  // oct of level l, or -1: coarser leaf
    }
  }
  // leaves of a refined level that touch a split cell of the same level (they receive deposits)
  for (int l = 1; l < s.nl; l++) {
    refined_lv_h[l].assign((size_t)(s.ncell[l] + 31) / 32, 0u);
    for (auto& kv : h->child_of[l]) refined_lv_h[l][kv.first >> 5] |= 1u << (kv.first & 31);
    CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.arefined[l], refined_lv_h[l].data(), refined_lv_h[l].size() * 4, cudaMemcpyHostToDevice, h->st));
    hasdep_h[l].assign((size_t)(s.ncell[l] + 31) / 32, 0u);
    for (auto& kv : h->child_of[l]) {
      const long long p = kv.first, po = p >> 3;
      const int k = (int)(p & 7);
      for (int a = 0; a < 3; a++)
        for (int side = 0; side < 2; side++) {
          long long q;
          if (side != ((k >> a) & 1)) q = (po << 3) | (k ^ (1 << a));
          else {
            const int no = nbo_h[l][po * 6 + 2 * a + side];
            if (no < 0) continue;
            q = ((long long)no << 3) | (k ^ (1 << a));
          }
          if (child_h[l][q] < 0) hasdep_h[l][q >> 5] |= 1u << (q & 31);
        }
    }
    CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.ahasdep[l], hasdep_h[l].data(), hasdep_h[l].size() * 4, cudaMemcpyHostToDevice, h->st));
  }
  // faces of refined cells towards a coarser leaf: (fine cell, coarse leaf, face), 4 per oct face
  for (int l = 1; l <= s.nl; l++) {
    for (long long o = 0; o < s.nocts[l]; o++)
      for (int f = 0; f < 6; f++) {
        const int pcell = nbr_h[l][o * 6 + f];
        if (pcell < 0) continue;
        const bool split = (l == 1) ? child0_h[pcell] >= 0 : child_h[l - 1][pcell] >= 0;
        if (split) continue;
        const int a = f >> 1, side = f & 1;
        // the six neighbours of the coarse leaf `pcell` on its own level l-1, for the ghost slopes (reading A21)
        for (int b = 0; b < 3; b++)
          for (int sd = 0; sd < 2; sd++) {
            long long q;                                                 // >= 0: cell of level l-1; else a code
            auto box = [&](int code) { const int bc = -1 - code; return bc == EMMA_RT_BC_INFLOW ? -5 : bc == EMMA_RT_BC_REFLECTIVE ? -2 - b : -1; };
            if (l == 1) { q = nb0(pcell, b, sd); if (q < 0) q = box((int)q); }
            else {
              const long long po = pcell >> 3;
              const int kk = pcell & 7, bit = (kk >> b) & 1;
              if (sd != bit) q = (po << 3) | (kk ^ (1 << b));
              else {
                const int pp = nbr_h[l - 1][po * 6 + 2 * b + sd];       // cell of level l-2
                if (pp < 0) q = box(pp);
                else {
                  const int ch = (l == 2) ? child0_h[pp] : child_h[l - 2][pp];
                  q = ch >= 0 ? (((long long)ch << 3) | (kk ^ (1 << b))) : (-16LL - pp);
                }
              }
            }
            slot_refs_h[l].push_back((int)q);
          }
        // the side's index (= its first list entry / 4) replaces the "coarser leaf" code -1 of the neighbour-oct table: the
        // cell kernels find their faces' records through it without another table
        nbo_h[l][o * 6 + f] = -16 - (int)(slot_cell_h[l].size() >> 2);
        for (int k = 0; k < 8; k++) {                                    // always 4 entries per oct side (kept aligned)
          if (((k >> a) & 1) != side) continue;
          if (l < s.nl && child_h[l][(o << 3) | k] >= 0)
            return fail(h, EMMA_RT_EINVAL, "resolution jump > 1 at oct %lld of level %d (PAPER.md:75)", o, l);
          slot_cell_h[l].push_back((int)((o << 3) | k));
          slot_coarse_h[l].push_back(pcell);
          slot_face_h[l].push_back((unsigned char)f);
        }
      }
    h->n_slots[l] = (int)slot_cell_h[l].size();
    CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.anbo[l], nbo_h[l].data(), nbo_h[l].size() * 4, cudaMemcpyHostToDevice, h->st));
    if (h->n_slots[l]) {
      CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.aslot_cell[l], slot_cell_h[l].data(), slot_cell_h[l].size() * 4, cudaMemcpyHostToDevice, h->st));
      CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.aslot_coarse[l], slot_coarse_h[l].data(), slot_coarse_h[l].size() * 4, cudaMemcpyHostToDevice, h->st));
      CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.aslot_face[l], slot_face_h[l].data(), slot_face_h[l].size(), cudaMemcpyHostToDevice, h->st));
      CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.aslot_refs[l], slot_refs_h[l].data(), slot_refs_h[l].size() * 4, cudaMemcpyHostToDevice, h->st));
    }
  }
  // level-0 leaves next to a split cell, with the mask of the faces that look at one (sorted by cell id)
  std::map<long long, unsigned> fix;
  for (auto& kv : h->child_of[0])
    for (int a = 0; a < 3; a++)
      for (int side = 0; side < 2; side++) {
        const long long q = nb0(kv.first, a, side);
        if (q < 0 || child0_h[q] >= 0) continue;
        fix[q] |= 1u << (2 * a + (1 - side));                   // q sees the split cell through its opposite face
      }
  for (auto& kv : fix) { fix_cell_h.push_back((int)kv.first); fix_mask_h.push_back((unsigned char)kv.second); }
  h->n_fix = (int)fix_cell_h.size();
  if (h->n_fix) {
    CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.afix_cell, fix_cell_h.data(), fix_cell_h.size() * 4, cudaMemcpyHostToDevice, h->st));
    CUDA_TRY(h, cudaMemcpyAsync(h->arena + h->lay.afix_mask, fix_mask_h.data(), fix_mask_h.size(), cudaMemcpyHostToDevice, h->st));
  }
  CUDA_TRY(h, cudaStreamSynchronize(h->st));   // the staging vectors above go out of scope
  return EMMA_RT_OK;
}

size_t field_elem_bytes(int field)
{
  switch (field) {
    case EMMA_RT_FIELD_U: return 16;
    case EMMA_RT_FIELD_F: return 12;
    default: return 4;
  }
}

// host -> library, one field of one level, through the scratch (= the inactive radiation buffer), chunked
int upload_field(emma_rt* h, int field, int level, int group, const void* src, bool src_is_device)
{
  const long long nc = h->sh.ncell[level];
  const size_t eb = field_elem_bytes(field);
  float4* Ug = (field == EMMA_RT_FIELD_U) ? h->Ulev(level) + (size_t)group * nc : nullptr;
  if (field == EMMA_RT_FIELD_U && h->sh.amr) h->amr_dirty = true;
  unsigned int* bad_dev = h->qcount() + 32;                            // invalid-value counter of the import kernel
  if (src_is_device) {
    // stream-ordered, no host wait: values are not validated here (a NaN stays a NaN and is reported by the next step)
    h->launches += launch_import(field, h->lv[level], Ug, (float)h->cfg.c_red_cm_s, 0, nc, src, nullptr, h->st);
    CUDA_TRY(h, cudaGetLastError());
    return EMMA_RT_OK;
  }
  char* scratch = (char*)h->U(1 - h->cur);
  const size_t cap = (size_t)h->sh.G * h->sh.ncell[0] * sizeof(float4);
  const long long chunk = (long long)(cap / eb);
  for (long long off = 0; off < nc; off += chunk) {
    const long long cnt = std::min(chunk, nc - off);
    CUDA_TRY(h, cudaMemcpyAsync(scratch, (const char*)src + (size_t)off * eb, (size_t)cnt * eb, cudaMemcpyHostToDevice, h->st));
    h->launches += launch_import(field, h->lv[level], Ug, (float)h->cfg.c_red_cm_s, off, cnt, scratch, bad_dev, h->st);
    CUDA_TRY(h, cudaGetLastError());
  }
  if (field == EMMA_RT_FIELD_U) {
    CUDA_TRY(h, cudaStreamSynchronize(h->st));
    return EMMA_RT_OK;
  }
  // n0 <= 0, T <= 0, x outside [0, 1] or anything non-finite would only surface as inf / NaN one step later: refuse now
  CUDA_TRY(h, cudaMemcpyAsync(&h->diag_pinned->err_last, bad_dev, 4, cudaMemcpyDeviceToHost, h->st));
  CUDA_TRY(h, cudaStreamSynchronize(h->st));
  const unsigned int n_bad = h->diag_pinned->err_last;
  if (n_bad) {
    CUDA_TRY(h, cudaMemsetAsync(bad_dev, 0, 4, h->st));
    return fail(h, EMMA_RT_EINVAL, "%u invalid value(s) in field %d of level %d (need finite n0 > 0, T > 0, 0 <= x <= 1)", n_bad, field, level);
  }
  return EMMA_RT_OK;
}

}  // namespace

namespace {

size_t arena_bytes_impl(const emma_rt_config* cfg, const emma_rt_amr* amr)
{
  Shape s;
  if (!make_shape(cfg, amr, s)) return 0;
  Layout L;
  make_layout(s, L);
  return L.total;
}

int init_impl(emma_rt** out, const emma_rt_config* cfg, const emma_rt_amr* amr, const emma_rt_fields* fields,
                 void* arena_dev, size_t arena_bytes)
{
  if (!out) return EMMA_RT_EINVAL;
  *out = nullptr;
  Shape s;
  if (!make_shape(cfg, amr, s) || !fields || !fields->n0 || !fields->x || !fields->T) return EMMA_RT_EINVAL;
  for (int l = 0; l <= s.nl; l++)
    if (!fields->n0[l] || !fields->x[l] || !fields->T[l]) return EMMA_RT_EINVAL;
  if (!arena_dev || ((uintptr_t)arena_dev % ALIGN) != 0) return EMMA_RT_EINVAL;
  emma_rt* h = new (std::nothrow) emma_rt();
  if (!h) return EMMA_RT_ENOMEM;
  h->cfg = *cfg; h->sh = s; h->err[0] = 0;
  make_layout(s, h->lay);
  h->arena = (char*)arena_dev;
  h->st = (cudaStream_t)cfg->stream;
  h->cur = 0; h->t_sim = 0; h->launches = 0; h->diag_pinned = nullptr; h->fused = 1; h->flux = EMMA_RT_FLUX_GLF; memset(h->inflow, 0, sizeof h->inflow);
  h->prof.st = h->st;
  h->dx = cfg->box_len_cm / s.n;
  *out = h;                                    // returned even on failure so the caller can read last_error
  if (arena_bytes < h->lay.total) return fail(h, EMMA_RT_ENOMEM, "arena too small: %zu < %zu", arena_bytes, h->lay.total);
  CUDA_TRY(h, cudaSetDevice(cfg->device));
  cudaDeviceProp prop;
  CUDA_TRY(h, cudaGetDeviceProperties(&prop, cfg->device));
  h->sm_count = prop.multiProcessorCount;
  // function attributes belong to the device's context: set them for every handle (a second handle on another GPU of the
  // same process needs its own), and take the occupancy of the persistent chemistry pass on THIS device
  CUDA_TRY(h, configure_transport_tma());
  CUDA_TRY(h, configure_transport_hll());
  CUDA_TRY(h, configure_fused(s.G));
  CUDA_TRY(h, configure_chemistry(s.G, &h->chem_ctas_per_sm));
  h->tune.nzc = env_int("EMMA_RT_TUNE_NZC", 0, 1, 4096);
  h->tune.nst = env_int("EMMA_RT_TUNE_NST", 6, 4, 8);
  if (h->tune.nst != 4 && h->tune.nst != 8) h->tune.nst = 6;
  h->tune.tma = env_int("EMMA_RT_TUNE_TMA", 1, 0, 1);
  h->tune.fused = env_int("EMMA_RT_TUNE_FUSED", 1, 0, 1);
  h->tune.chem_ctas = env_int("EMMA_RT_TUNE_CHEMCTAS", 0, 1, 32);
  if (h->tune.chem_ctas > 0) h->chem_ctas_per_sm = h->tune.chem_ctas;
  CUDA_TRY(h, cudaMallocHost((void**)&h->diag_pinned, sizeof(DiagDev)));
  for (int b = 0; b < 2; b++) {
    const int r = make_transport_maps(h->U(b), s.n, s.G, &h->tmaps[b]);
    if (r != 0) return fail(h, EMMA_RT_ECUDA, "cuTensorMapEncodeTiled failed (%d)", r);
    const int rh = make_transport_maps(h->U(b), s.n, s.G, &h->tmaps_h[b], 16, hll_tile_x(), hll_main_x());
    if (rh != 0) return fail(h, EMMA_RT_ECUDA, "cuTensorMapEncodeTiled failed (%d)", rh);
    const int rf = make_transport_maps(h->U(b), s.n, s.G, &h->tmaps_f[b], fused_tile_y());
    if (rf != 0) return fail(h, EMMA_RT_ECUDA, "cuTensorMapEncodeTiled failed (%d)", rf);
  }

  // ---- AMR index arrays (a-0: per-level oct arrays with parent / coarse-ancestor / child indices)
  std::vector<std::vector<int>> parent_h(s.nl + 1), child_h(s.nl + 1);
  for (int l = 1; l <= s.nl; l++) {
    parent_h[l].resize(s.nocts[l]);
    h->anc0_h[l].resize(s.nocts[l]);
    for (long long o = 0; o < s.nocts[l]; o++) {
      const long long p = amr->parent[l - 1][o];
      if (p < 0 || p >= s.ncell[l - 1]) return fail(h, EMMA_RT_EINVAL, "parent[%d][%lld] out of range", l - 1, o);
      if (!h->child_of[l - 1].emplace(p, (int)o).second) return fail(h, EMMA_RT_EINVAL, "cell split twice on level %d", l - 1);
      parent_h[l][o] = (int)p;
      h->anc0_h[l][o] = (l == 1) ? (int)p : h->anc0_h[l - 1][p >> 3];
    }
  }
  CUDA_TRY(h, cudaMemsetAsync(h->arena, 0, h->lay.total, h->st));
  for (int l = 0; l <= s.nl; l++) {
    LevelDev& L = h->lv[l];
    memset(&L, 0, sizeof L);
    L.ncell = s.ncell[l]; L.nocts = s.nocts[l];
    L.n0 = (float*)(h->arena + h->lay.n0[l]); L.xs = (float*)(h->arena + h->lay.xs[l]); L.eps = (float*)(h->arena + h->lay.eps[l]);
    L.subc = s.record ? (unsigned int*)(h->arena + h->lay.subc[l]) : nullptr;
    L.srcmask = (unsigned int*)(h->arena + h->lay.srcmask[l]);
    L.src_cell = (int*)(h->arena + h->lay.src_cell[l]);
    L.src_S = (float*)(h->arena + h->lay.src_S[l]);
    L.n_src = 0;
    const double dxl = h->dx / (double)(1 << l);
    L.dV = dxl * dxl * dxl;
    L.dV_total = L.dV;
    if (l >= 1) {
      L.parent = (int*)(h->arena + h->lay.parent[l]);
      L.anc0 = (int*)(h->arena + h->lay.anc0[l]);
      CUDA_TRY(h, cudaMemcpyAsync(L.parent, parent_h[l].data(), s.nocts[l] * 4, cudaMemcpyHostToDevice, h->st));
      CUDA_TRY(h, cudaMemcpyAsync(L.anc0, h->anc0_h[l].data(), s.nocts[l] * 4, cudaMemcpyHostToDevice, h->st));
      if (l < s.nl) {
        L.child = (int*)(h->arena + h->lay.child[l]);
        child_h[l].assign(s.ncell[l], -1);
        for (auto& kv : h->child_of[l]) child_h[l][kv.first] = kv.second;
        CUDA_TRY(h, cudaMemcpyAsync(L.child, child_h[l].data(), s.ncell[l] * 4, cudaMemcpyHostToDevice, h->st));
      }
      if (l >= 2) L.Ut = (float4*)(h->arena + h->lay.Ut[l]);
    }
  }
  std::vector<unsigned int> refined_h;
  if (s.nl > 0) {
    h->lv[0].refined = (unsigned int*)(h->arena + h->lay.refined0);
    refined_h.assign((size_t)(s.ncell[0] + 31) / 32, 0u);
    for (auto& kv : h->child_of[0]) refined_h[kv.first >> 5] |= 1u << (kv.first & 31);
    CUDA_TRY(h, cudaMemcpyAsync(h->lv[0].refined, refined_h.data(), refined_h.size() * 4, cudaMemcpyHostToDevice, h->st));
  }
  // ---- standard AMR transport (A21): oct neighbour pointers and the index arrays derived from them
  h->n_fix = 0; h->amr_dirty = false;
  for (int l = 0; l <= MAXL; l++) { h->acur[l] = 0; h->n_slots[l] = 0; }
  if (s.amr) {
    const int rc_topo = init_amr_topology(h, parent_h, child_h);
    if (rc_topo != EMMA_RT_OK) return rc_topo;
  }
  CUDA_TRY(h, cudaStreamSynchronize(h->st));   // host staging vectors go out of scope below

  // ---- fields: N0, X, T (-> eps, A10) per level; U0 per group; then the children means of split cells (A14)
  int rc;
  for (int l = 0; l <= s.nl; l++) {
    if ((rc = upload_field(h, EMMA_RT_FIELD_N0, l, 0, fields->n0[l], false)) != EMMA_RT_OK) return rc;
    if ((rc = upload_field(h, EMMA_RT_FIELD_X, l, 0, fields->x[l], false)) != EMMA_RT_OK) return rc;
    if ((rc = upload_field(h, EMMA_RT_FIELD_T, l, 0, fields->T[l], false)) != EMMA_RT_OK) return rc;
  }
  if (fields->U0)
    for (int g = 0; g < s.G; g++)
      if (fields->U0[g] && (rc = upload_field(h, EMMA_RT_FIELD_U, 0, g, fields->U0[g], false)) != EMMA_RT_OK) return rc;
  for (int l = s.nl; l >= 1; l--) h->launches += launch_restrict_init(h->lv, l, h->st);
  if (s.amr) {                                 // refined cells start with their parent's radiation
    const AmrDev A = amr_view(h);
    for (int l = 1; l <= s.nl; l++) h->launches += launch_amr_inject_init(h->lv[l], A, l, h->st);
  }
  CUDA_TRY(h, cudaGetLastError());
  CUDA_TRY(h, cudaStreamSynchronize(h->st));
  return EMMA_RT_OK;
}

int set_sources_impl(emma_rt* h, int64_t n_src, const double* pos, const double* Q)
{
  if (!h) return EMMA_RT_EINVAL;
  const Shape& s = h->sh;
  if (n_src < 0 || (n_src > 0 && (!pos || !Q))) return fail(h, EMMA_RT_EINVAL, "bad source arguments");
  for (int64_t i = 0; i < n_src; i++) {
    for (int k = 0; k < 3; k++)
      if (!(pos[3 * i + k] >= 0.0 && pos[3 * i + k] < 1.0)) return fail(h, EMMA_RT_EINVAL, "source %lld outside the box", (long long)i);
    for (int g = 0; g < s.G; g++)
      if (!(Q[i * s.G + g] >= 0.0) || std::isinf(Q[i * s.G + g])) return fail(h, EMMA_RT_EINVAL, "source %lld: bad Q", (long long)i);
  }
  // A12: NGP into the leaf containing the position; S_g = Q_g / dV_leaf; same-cell sources add (in fp64)
  std::map<long long, std::vector<double>> per_level[MAXL + 1];
  for (int64_t i = 0; i < n_src; i++) {
    const double fx = pos[3 * i] * s.n, fy = pos[3 * i + 1] * s.n, fz = pos[3 * i + 2] * s.n;
    int ix = std::min((int)std::floor(fx), s.n - 1), iy = std::min((int)std::floor(fy), s.n - 1), iz = std::min((int)std::floor(fz), s.n - 1);
    double ox = fx - ix, oy = fy - iy, oz = fz - iz;
    int lvl = 0;
    long long cell = ix + (long long)s.n * (iy + (long long)s.n * iz);
    if (h->cfg.chemistry || s.amr) {             // CRTA with chemistry off: sources are folded to the coarse cell (A9)
      while (lvl < s.nl) {
        auto it = h->child_of[lvl].find(cell);
        if (it == h->child_of[lvl].end()) break;
        const int cx = ox >= 0.5, cy = oy >= 0.5, cz = oz >= 0.5;
        ox = 2 * ox - cx; oy = 2 * oy - cy; oz = 2 * oz - cz;
        cell = 8LL * it->second + (cx + 2 * cy + 4 * cz);
        lvl++;
      }
    }
    auto& v = per_level[lvl][cell];
    if (v.empty()) v.assign(s.G, 0.0);
    for (int g = 0; g < s.G; g++) v[g] += Q[i * s.G + g] / h->lv[lvl].dV;
  }
  for (int l = 0; l <= s.nl; l++)
    if ((long long)per_level[l].size() > s.max_src) return fail(h, EMMA_RT_EINVAL, "more than max_source_cells source cells");
  CUDA_TRY(h, cudaStreamSynchronize(h->st));
  for (int l = 0; l <= s.nl; l++) {
    LevelDev& L = h->lv[l];
    std::vector<int> cells;
    std::vector<float> S;
    for (auto& kv : per_level[l]) {
      cells.push_back((int)kv.first);
      for (int g = 0; g < s.G; g++) S.push_back((float)kv.second[g]);
    }
    CUDA_TRY(h, cudaMemsetAsync(L.srcmask, 0, (size_t)(L.ncell + 31) / 32 * 4, h->st));
    L.n_src = (int)cells.size();
    if (L.n_src) {
      CUDA_TRY(h, cudaMemcpyAsync(L.src_cell, cells.data(), cells.size() * 4, cudaMemcpyHostToDevice, h->st));
      CUDA_TRY(h, cudaMemcpyAsync(L.src_S, S.data(), S.size() * 4, cudaMemcpyHostToDevice, h->st));
      h->launches += launch_set_bits(L.srcmask, L.src_cell, L.n_src, h->st);
      CUDA_TRY(h, cudaGetLastError());
    }
    CUDA_TRY(h, cudaStreamSynchronize(h->st));
  }
  return EMMA_RT_OK;
}

// geometry- and physics-constants of one step of size dt (everything but the z-chunking of a particular kernel)
void base_params(const emma_rt* h, double dt, TransportParams& tp, ChemParams& cp, bool& any_inflow)
{
  const Shape& s = h->sh;
  const double c = h->cfg.c_red_cm_s;
  tp.n = s.n; tp.G = s.G;
  any_inflow = false;
  for (int f = 0; f < 6; f++) { tp.bc[f] = h->cfg.bc[f]; any_inflow = any_inflow || h->cfg.bc[f] == EMMA_RT_BC_INFLOW; }
  memcpy(tp.inflow, h->inflow, sizeof tp.inflow);
  tp.tiles_x = (s.n + 31) / 32; tp.tiles_y = (s.n + 15) / 16;
  tp.z_lo = 0; tp.z_hi = s.n;
  tp.zchunk = s.n; tp.nzc = 1;
  tp.nst = h->tune.nst;
  tp.pf = 2;
  tp.want_total = h->cfg.chemistry ? 0 : 1;
  tp.nu = (float)(c * dt / h->dx);
  tp.c0 = (float)(1.0 - 3.0 * (c * dt / h->dx));
  tp.c1 = (float)(0.5 * (c * dt / h->dx));
  tp.dV = h->lv[0].dV;
  memset(&cp, 0, sizeof cp);
  cp.G = s.G; cp.otsa = h->cfg.otsa; cp.thermal = h->cfg.thermal; cp.max_halvings = h->cfg.max_halvings;
  cp.record = s.record ? 1 : 0;
  cp.dt = (float)dt; cp.e_tol = (float)h->cfg.e_tol;
  for (int g = 0; g < s.G; g++) {
    cp.csig[g] = (float)(c * h->cfg.sigma_N[g]);
    cp.csigE[g] = (float)(c * (h->cfg.sigma_E[g] * h->cfg.E_mean[g] - h->cfg.sigma_N[g] * E_HI_ERG));
  }
}

int step_impl(emma_rt* h, double dt, int32_t n_steps, emma_rt_diag* diag_last)
{
  if (!h) return EMMA_RT_EINVAL;
  if (!(dt > 0.0) || n_steps < 0) return fail(h, EMMA_RT_EINVAL, "dt must be > 0 and n_steps >= 0");
  const Shape& s = h->sh;
  const double c = h->cfg.c_red_cm_s;
  if (3.0 * c * dt > h->dx * (1.0 + 1e-12)) return fail(h, EMMA_RT_ECFL, "dt = %g exceeds dx/(3 c) = %g (A4)", dt, h->dx / (3 * c));

  TransportParams tp;
  ChemParams cp;
  bool any_inflow = false;
  base_params(h, dt, tp, cp, any_inflow);
  // z chunks.  Every CTA costs (its planes + ~3 planes of prologue) and the SMs hold `per_sm` CTAs each, so a launch
  // takes ceil(blocks / (per_sm SMs)) rounds of (zchunk + 3) plane-times: pick the chunk count that minimises that
  // (at 512^3 x 3 one chunk per column is 1536 CTAs = 5.19 rounds, i.e. 14 % of the last round idle).
  auto pick_zchunks = [&](TransportParams& q, int per, int per_sm) -> bool {
    const long long slots = (long long)per_sm * h->sm_count;
    int best = 1; double best_cost = 1e300;
    const int env_nzc = h->tune.nzc;
    for (int nzc = 1; nzc <= std::max(1, s.n / 8); nzc++) {
      const int zc = (s.n + nzc - 1) / nzc;
      const int nz = (s.n + zc - 1) / zc;
      if (nz != nzc) continue;
      const long long blocks = (long long)per * nz;
      if (blocks > TRANSPORT_MAX_BLOCKS) break;
      const double cost = (double)((blocks + slots - 1) / slots) * (zc + 3);
      if (cost < best_cost * (1.0 - 1e-9)) { best_cost = cost; best = nzc; }
    }
    // the override applies to every dense pass whose partial-sum slots it fits (a pass that is not even used must not refuse the step)
    if (env_nzc > 0 && env_nzc <= s.n && (long long)per * env_nzc <= TRANSPORT_MAX_BLOCKS) best = env_nzc;
    q.zchunk = (s.n + best - 1) / best;
    q.nzc = (s.n + q.zchunk - 1) / q.zchunk;
    return (long long)per * q.nzc <= TRANSPORT_MAX_BLOCKS;
  };
  if (!pick_zchunks(tp, tp.tiles_x * tp.tiles_y * s.G, 2)) return fail(h, EMMA_RT_EINVAL, "grid too large for the partial-sum slots");
  const bool use_tma = !any_inflow && h->tune.tma != 0;

  // fused schedule (fused.cu): all G groups of a tile in one CTA, one CTA per SM
  const bool hll = h->flux == EMMA_RT_FLUX_HLL;
  TransportParams hp = tp;                     // HLL pass (transport_hll.cu): one group per CTA, 31-cell-wide tiles
  hp.tiles_x = (s.n + hll_tile_x() - 1) / hll_tile_x();
  if (hll && !pick_zchunks(hp, hp.tiles_x * hp.tiles_y * s.G, hll_ctas_per_sm())) return fail(h, EMMA_RT_EINVAL, "grid too large for the partial-sum slots");
  const bool fused = !hll && !any_inflow && h->cfg.chemistry && h->fused && h->tune.fused != 0;
  TransportParams fp = tp;
  fp.tiles_y = (s.n + fused_tile_y() - 1) / fused_tile_y();
  if (fused && !pick_zchunks(fp, fp.tiles_x * fp.tiles_y, fused_ctas_per_sm())) return fail(h, EMMA_RT_EINVAL, "grid too large for the partial-sum slots");

  if (s.amr) {
    const int rc = step_amr(h, dt, n_steps, tp, hp, cp, use_tma, hll);
    if (rc != EMMA_RT_OK) return rc;
  }
  for (int step = 0; step < (s.amr ? 0 : n_steps); step++) {
    int off = 0, np = 0;
    Partial* P = h->parts();
    if (fused) {
      // 1+3. transport and the first chemistry trip of every unrefined coarse cell in one pass; then the compacted
      // tail, then CRTA on the refined cells (they read the U* this pass wrote into their coarse ancestors)
      float4* U = h->U(1 - h->cur);
      h->prof.begin(EMMA_RT_K_FUSED);
      const int k = launch_fused(fp, h->tmaps_f[h->cur], U, cp, h->lv[0], (int*)(h->arena + h->lay.queue), h->qcount(), P + off, &np, h->st);
      if (!k) return fail(h, EMMA_RT_ECUDA, "fused launch failed: %s", cudaGetErrorString(cudaGetLastError()));
      h->prof.end();
      h->launches += k;
      off += np;
      h->cur = 1 - h->cur;
      h->launches += launch_chem_tail(cp, h->lv[0], U, s.ncell[0], (int*)(h->arena + h->lay.queue), h->qcount(), P + off, &np,
                                      h->sm_count, h->st, &h->prof);
      off += np;
      for (int l = s.nl; l >= 1; l--) {
        h->prof.begin(EMMA_RT_K_CHEM_REFINED);
        h->launches += launch_chem_refined(cp, h->lv, l, s.nl, U, s.ncell[0], h->crta_queue(l), P + off, &np, h->sm_count, h->st);
        h->prof.end();
        off += np;
      }
      h->t_sim += dt;
      h->prof.begin(EMMA_RT_K_FINALIZE);
      h->launches += launch_finalize(P, off, h->diag(), h->qcount(), h->t_sim, h->st);
      h->prof.end();
      continue;
    }
    // 1. coarse transport, old buffer -> new buffer (Jacobi)
    h->prof.begin(EMMA_RT_K_TRANSPORT);
    if (hll) {
      const int k = launch_transport_hll(hp, h->tmaps_h[h->cur], h->U(1 - h->cur), P + off, &np, h->st);
      if (!k) return fail(h, EMMA_RT_ECUDA, "HLL transport launch failed: %s", cudaGetErrorString(cudaGetLastError()));
      h->launches += k;
    } else if (use_tma) {
      const int k = launch_transport_tma(tp, h->tmaps[h->cur], h->U(1 - h->cur), P + off, &np, h->st);
      if (!k) return fail(h, EMMA_RT_ECUDA, "transport launch failed: %s", cudaGetErrorString(cudaGetLastError()));
      h->launches += k;
    } else {
      h->launches += launch_transport(tp, h->U(h->cur), h->U(1 - h->cur), P + off, &np, h->st);
    }
    h->prof.end();
    off += np;
    h->cur = 1 - h->cur;
    float4* U = h->U(h->cur);
    if (h->cfg.chemistry) {
      // 2-4. CRTA: deepest refined level first (inject -> leaf chemistry -> restrict), then the unrefined coarse cells
      for (int l = s.nl; l >= 1; l--) {
        h->prof.begin(EMMA_RT_K_CHEM_REFINED);
        h->launches += launch_chem_refined(cp, h->lv, l, s.nl, U, s.ncell[0], h->crta_queue(l), P + off, &np, h->sm_count, h->st);
        h->prof.end();
        off += np;
      }
      h->launches += launch_chem_level0(cp, h->lv[0], U, s.ncell[0], (int*)(h->arena + h->lay.queue), h->qcount(),
                                        P + off, &np, h->sm_count, h->chem_ctas_per_sm, h->st, &h->prof);
      off += np;
    } else {
      h->prof.begin(EMMA_RT_K_OTHER);
      h->launches += launch_inject_sources(h->lv[0], s.G, (float)dt, U, s.ncell[0], P + off, &np, h->st);
      h->prof.end();
      off += np;
    }
    h->t_sim += dt;
    // 5. diagnostics
    h->prof.begin(EMMA_RT_K_FINALIZE);
    h->launches += launch_finalize(P, off, h->diag(), h->qcount(), h->t_sim, h->st);
    h->prof.end();
  }
  CUDA_TRY(h, cudaGetLastError());
  if (!diag_last) return EMMA_RT_OK;
  if (n_steps == 0) {                          // state query: photons currently in the box (summed on the device)
    memset(diag_last, 0, sizeof *diag_last);
    diag_last->t_sim = h->t_sim;
    diag_last->dtau_min = INFINITY;
    double* tot_dev = (double*)(h->qcount() + 16);                     // scratch double inside the counter block
    h->launches += launch_sum_N(h->U(h->cur), (long long)s.G * s.ncell[0], h->lv[0].dV, h->parts(), tot_dev, h->st);
    CUDA_TRY(h, cudaGetLastError());
    CUDA_TRY(h, cudaMemcpyAsync(&h->diag_pinned->d.photons_total, tot_dev, sizeof(double), cudaMemcpyDeviceToHost, h->st));
    CUDA_TRY(h, cudaStreamSynchronize(h->st));
    diag_last->photons_total = h->diag_pinned->d.photons_total;
    return EMMA_RT_OK;
  }
  CUDA_TRY(h, cudaMemcpyAsync(h->diag_pinned, h->diag(), sizeof(DiagDev), cudaMemcpyDeviceToHost, h->st));
  CUDA_TRY(h, cudaStreamSynchronize(h->st));
  *diag_last = h->diag_pinned->d;
  if (h->diag_pinned->d.n_nonfinite > 0) return fail(h, EMMA_RT_ENONFINITE, "%lld non-finite cells", (long long)h->diag_pinned->d.n_nonfinite);
  if (h->diag_pinned->err_last & 1u) return fail(h, EMMA_RT_ESUBCYCLE, "sub-cycle guard hit (max_halvings or %d sub-steps)", EMMA_RT_MAX_SUBSTEPS);
  return EMMA_RT_OK;
}

// One coupled step for a caller whose state lives in HOST memory (include/emma_rt.h: emma_rt_step_host).  Same kernels
// and arithmetic as write(U, X, T) -> step(dt, 1) -> read(U, X, T), but the grid goes through the device in z-slabs on
// three streams, so the upload of slab k+1, the fused pass over slab k and the download of slab k-1 overlap: both copy
// engines are busy at once (PCIe is full duplex) and the compute hides behind them.  The paper's own GPU engines spent
// ~70 % of their time in exactly this traffic.
int step_host_impl(emma_rt* h, double dt, const emma_rt_host_state* in, const emma_rt_host_state* out, emma_rt_diag* diag_last)
{
  if (!h || !in || !out || !in->U || !in->x || !in->T || !out->U || !out->x || !out->T) return EMMA_RT_EINVAL;
  const Shape& s = h->sh;
  const double c = h->cfg.c_red_cm_s;
  if (!(dt > 0.0)) return fail(h, EMMA_RT_EINVAL, "dt must be > 0");
  if (3.0 * c * dt > h->dx * (1.0 + 1e-12)) return fail(h, EMMA_RT_ECFL, "dt = %g exceeds dx/(3 c) = %g (A4)", dt, h->dx / (3 * c));
  for (int g = 0; g < s.G; g++)
    if (!in->U[g] || !out->U[g]) return fail(h, EMMA_RT_EINVAL, "NULL radiation array of group %d", g);
  TransportParams tp;
  ChemParams cp;
  bool any_inflow = false;
  base_params(h, dt, tp, cp, any_inflow);
  if (s.slab_planes == 0 || any_inflow || h->flux != EMMA_RT_FLUX_GLF || !h->fused || !h->tune.fused)
    return fail(h, EMMA_RT_ESTATE, "emma_rt_step_host needs a uniform grid, chemistry on, the GLF flux, the fused schedule and no inflow face");
  tp.tiles_y = (s.n + fused_tile_y() - 1) / fused_tile_y();
  const int nblk = tp.tiles_x * tp.tiles_y;                            // one CTA per tile column and slab
  const int tail_blocks = std::min(h->sm_count * 8, MAX_PART_BLOCKS);
  int zs = s.slab_planes;
  while ((long long)((s.n + zs - 1) / zs) * (nblk + tail_blocks) > PART_SLOTS && zs < s.n) zs *= 2;   // fewer, thicker slabs
  // thicker slabs than the staging area holds are never needed for n <= 1290 (41 x 81 tiles x 32 slabs fit the slots)
  if (zs > s.slab_planes) return fail(h, EMMA_RT_EINVAL, "grid too large for the partial-sum slots");
  const int K = (s.n + zs - 1) / zs;
  if (!h->s_in) {
    CUDA_TRY(h, cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking));
    CUDA_TRY(h, cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking));
    CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_start, cudaEventDisableTiming));
  }
  while ((int)h->ev_in.size() < K) {
    cudaEvent_t a, b;
    CUDA_TRY(h, cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
    CUDA_TRY(h, cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
    h->ev_in.push_back(a); h->ev_c.push_back(b);
  }
  const size_t plane = (size_t)s.n * s.n;
  const float cr = (float)c;
  LevelDev& L0 = h->lv[0];
  float4* Uold = h->U(h->cur);
  float4* Unew = h->U(1 - h->cur);
  unsigned int* bad_dev = h->qcount() + 32;
  char* stage = h->arena + h->lay.host_stage;
  auto z_lo = [&](int k) { return k * zs; };
  auto z_hi = [&](int k) { return std::min(s.n, (k + 1) * zs); };

  // the copy streams start after whatever the caller's stream still has in flight on this state
  CUDA_TRY(h, cudaEventRecord(h->ev_start, h->st));
  CUDA_TRY(h, cudaStreamWaitEvent(h->s_in, h->ev_start, 0));
  CUDA_TRY(h, cudaStreamWaitEvent(h->s_out, h->ev_start, 0));

  // ---- uploads, in the order the compute needs them: slab 0 reads the last plane of slab K-1 (periodic z), so K-1 goes
  // first.  Raw bytes land in the state arrays themselves and are converted in place (F -> F/c, x -> code, T -> e/n0).
  auto upload = [&](int k) -> int {
    const size_t off = (size_t)z_lo(k) * plane, cnt = (size_t)(z_hi(k) - z_lo(k)) * plane;
    for (int g = 0; g < s.G; g++) {
      float4* Ug = Uold + (size_t)g * s.ncell[0];
      CUDA_TRY(h, cudaMemcpyAsync(Ug + off, in->U[g] + 4 * off, cnt * 16, cudaMemcpyHostToDevice, h->s_in));
      h->launches += launch_import(EMMA_RT_FIELD_U, L0, Ug, cr, (long long)off, (long long)cnt, Ug + off, nullptr, h->s_in);
    }
    CUDA_TRY(h, cudaMemcpyAsync(L0.xs + off, in->x + off, cnt * 4, cudaMemcpyHostToDevice, h->s_in));
    h->launches += launch_import(EMMA_RT_FIELD_X, L0, nullptr, cr, (long long)off, (long long)cnt, L0.xs + off, bad_dev, h->s_in);
    CUDA_TRY(h, cudaMemcpyAsync(L0.eps + off, in->T + off, cnt * 4, cudaMemcpyHostToDevice, h->s_in));
    h->launches += launch_import(EMMA_RT_FIELD_T, L0, nullptr, cr, (long long)off, (long long)cnt, L0.eps + off, bad_dev, h->s_in);
    CUDA_TRY(h, cudaEventRecord(h->ev_in[k], h->s_in));
    return EMMA_RT_OK;
  };
  int rc;
  if (K > 1 && (rc = upload(K - 1)) != EMMA_RT_OK) return rc;
  for (int k = 0; k < (K > 1 ? K - 1 : 1); k++)
    if ((rc = upload(k)) != EMMA_RT_OK) return rc;

  // ---- per slab: fused pass + tail on the caller's stream once its three input slabs are there; export + download behind it
  int off_parts = 0;
  Partial* P = h->parts();
  int* queue = (int*)(h->arena + h->lay.queue);
  for (int k = 0; k < K; k++) {
    for (int q : {(k + K - 1) % K, k, (k + 1) % K}) CUDA_TRY(h, cudaStreamWaitEvent(h->st, h->ev_in[q], 0));
    TransportParams fp = tp;
    fp.z_lo = z_lo(k); fp.z_hi = z_hi(k);
    fp.zchunk = fp.z_hi - fp.z_lo; fp.nzc = 1;
    int np = 0;
    h->prof.begin(EMMA_RT_K_FUSED);
    const int kf = launch_fused(fp, h->tmaps_f[h->cur], Unew, cp, L0, queue, h->qcount(), P + off_parts, &np, h->st);
    if (!kf) return fail(h, EMMA_RT_ECUDA, "fused launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    h->prof.end();
    h->launches += kf;
    off_parts += np;
    if (cp.thermal) {
      h->launches += launch_chem_tail(cp, L0, Unew, s.ncell[0], queue, h->qcount(), P + off_parts, &np, h->sm_count, h->st, &h->prof);
      off_parts += np;
      CUDA_TRY(h, cudaMemsetAsync(h->qcount(), 0, 8, h->st));           // queue counters of the next slab
    }
    CUDA_TRY(h, cudaEventRecord(h->ev_c[k], h->st));
    // download: everything on s_out is in order, so the one staging slab is free again when the next export starts
    CUDA_TRY(h, cudaStreamWaitEvent(h->s_out, h->ev_c[k], 0));
    const size_t off = (size_t)z_lo(k) * plane, cnt = (size_t)(z_hi(k) - z_lo(k)) * plane;
    char* sp = stage;
    for (int g = 0; g < s.G; g++, sp += cnt * 16) {
      h->launches += launch_export(EMMA_RT_FIELD_U, L0, Unew + (size_t)g * s.ncell[0], cr, (long long)off, (long long)cnt, sp, h->s_out);
      CUDA_TRY(h, cudaMemcpyAsync(out->U[g] + 4 * off, sp, cnt * 16, cudaMemcpyDeviceToHost, h->s_out));
    }
    h->launches += launch_export(EMMA_RT_FIELD_X, L0, nullptr, cr, (long long)off, (long long)cnt, sp, h->s_out);
    CUDA_TRY(h, cudaMemcpyAsync(out->x + off, sp, cnt * 4, cudaMemcpyDeviceToHost, h->s_out));
    sp += cnt * 4;
    h->launches += launch_export(EMMA_RT_FIELD_T, L0, nullptr, cr, (long long)off, (long long)cnt, sp, h->s_out);
    CUDA_TRY(h, cudaMemcpyAsync(out->T + off, sp, cnt * 4, cudaMemcpyDeviceToHost, h->s_out));
  }
  h->cur = 1 - h->cur;
  h->t_sim += dt;
  h->prof.begin(EMMA_RT_K_FINALIZE);
  h->launches += launch_finalize(P, off_parts, h->diag(), h->qcount(), h->t_sim, h->st);
  h->prof.end();
  CUDA_TRY(h, cudaGetLastError());
  CUDA_TRY(h, cudaMemcpyAsync(h->diag_pinned, h->diag(), sizeof(DiagDev), cudaMemcpyDeviceToHost, h->st));
  CUDA_TRY(h, cudaMemcpyAsync(&h->diag_pinned->pad_bad, bad_dev, 4, cudaMemcpyDeviceToHost, h->st));
  CUDA_TRY(h, cudaStreamSynchronize(h->s_in));
  CUDA_TRY(h, cudaStreamSynchronize(h->st));
  CUDA_TRY(h, cudaStreamSynchronize(h->s_out));
  if (h->diag_pinned->pad_bad) {
    const unsigned int n_bad = h->diag_pinned->pad_bad;
    CUDA_TRY(h, cudaMemsetAsync(bad_dev, 0, 4, h->st));
    return fail(h, EMMA_RT_EINVAL, "%u invalid value(s) in the host state (need finite T > 0, 0 <= x <= 1)", n_bad);
  }
  if (diag_last) *diag_last = h->diag_pinned->d;
  if (h->diag_pinned->d.n_nonfinite > 0) return fail(h, EMMA_RT_ENONFINITE, "%lld non-finite cells", (long long)h->diag_pinned->d.n_nonfinite);
  if (h->diag_pinned->err_last & 1u) return fail(h, EMMA_RT_ESUBCYCLE, "sub-cycle guard hit (max_halvings or %d sub-steps)", EMMA_RT_MAX_SUBSTEPS);
  return EMMA_RT_OK;
}

int read_impl(emma_rt* h, int32_t field, int32_t level, int32_t group, void* dst, size_t bytes, int32_t dst_is_device)
{
  if (!h || !dst) return EMMA_RT_EINVAL;
  const Shape& s = h->sh;
  if (level < 0 || level > s.nl) return fail(h, EMMA_RT_EINVAL, "level out of range");
  if (field < EMMA_RT_FIELD_U || field > EMMA_RT_FIELD_XNEUTRAL) return fail(h, EMMA_RT_EINVAL, "unknown field");
  const bool rad = field == EMMA_RT_FIELD_U || field == EMMA_RT_FIELD_N || field == EMMA_RT_FIELD_F;
  if (rad && ((level != 0 && !s.amr) || group < 0 || group >= s.G)) return fail(h, EMMA_RT_EINVAL, "radiation fields live on level 0 (every level with amr_transport), group in range");
  if (field == EMMA_RT_FIELD_SUBCYCLES && !s.record) return fail(h, EMMA_RT_ESTATE, "record_subcycles was not set");
  const long long nc = s.ncell[level];
  const size_t eb = field_elem_bytes(field);
  if (bytes != (size_t)nc * eb) return fail(h, EMMA_RT_EINVAL, "size mismatch: %zu != %zu", bytes, (size_t)nc * eb);
  const float4* Ug = rad ? h->Ulev(level) + (size_t)group * nc : nullptr;
  const float cr = (float)h->cfg.c_red_cm_s;
  if (dst_is_device) {
    h->launches += launch_export(field, h->lv[level], Ug, cr, 0, nc, dst, h->st);
    CUDA_TRY(h, cudaGetLastError());
    return EMMA_RT_OK;
  }
  char* scratch = (char*)h->U(1 - h->cur);
  const size_t cap = (size_t)s.G * s.ncell[0] * sizeof(float4);
  const long long chunk = (long long)(cap / eb);
  for (long long off = 0; off < nc; off += chunk) {
    const long long cnt = std::min(chunk, nc - off);
    h->launches += launch_export(field, h->lv[level], Ug, cr, off, cnt, scratch, h->st);
    CUDA_TRY(h, cudaGetLastError());
    CUDA_TRY(h, cudaMemcpyAsync((char*)dst + (size_t)off * eb, scratch, (size_t)cnt * eb, cudaMemcpyDeviceToHost, h->st));
    CUDA_TRY(h, cudaStreamSynchronize(h->st));
  }
  return EMMA_RT_OK;
}

int write_impl(emma_rt* h, int32_t field, int32_t level, int32_t group, const void* src, size_t bytes, int32_t src_is_device)
{
  if (!h || !src) return EMMA_RT_EINVAL;
  const Shape& s = h->sh;
  if (level < 0 || level > s.nl) return fail(h, EMMA_RT_EINVAL, "level out of range");
  if (field != EMMA_RT_FIELD_U && field != EMMA_RT_FIELD_X && field != EMMA_RT_FIELD_T && field != EMMA_RT_FIELD_N0)
    return fail(h, EMMA_RT_EINVAL, "field is not writable");
  if (field == EMMA_RT_FIELD_U && ((level != 0 && !s.amr) || group < 0 || group >= s.G)) return fail(h, EMMA_RT_EINVAL, "U lives on level 0 (every level with amr_transport), group in range");
  const size_t eb = field_elem_bytes(field);
  if (bytes != (size_t)s.ncell[level] * eb) return fail(h, EMMA_RT_EINVAL, "size mismatch");
  return upload_field(h, field, level, group, src, src_is_device != 0);
}

int profile_impl(emma_rt* h, int32_t enable, double* ms_out, int64_t* launches_out)
{
  if (!h) return EMMA_RT_EINVAL;
  CUDA_TRY(h, cudaStreamSynchronize(h->st));
  double ms[EMMA_RT_K_COUNT] = {0};
  int64_t cnt[EMMA_RT_K_COUNT] = {0};
  for (const Profiler::Span& sp : h->prof.spans) {
    float t = 0.f;
    CUDA_TRY(h, cudaEventElapsedTime(&t, sp.a, sp.b));
    ms[sp.kind] += t;
    cnt[sp.kind]++;
  }
  for (int k = 0; k < EMMA_RT_K_COUNT; k++) {
    if (ms_out) ms_out[k] = ms[k];
    if (launches_out) launches_out[k] = cnt[k];
  }
  h->prof.reset();
  h->prof.on = enable != 0;
  return EMMA_RT_OK;
}

}  // namespace

extern "C" {

size_t emma_rt_arena_bytes(const emma_rt_config* cfg, const emma_rt_amr* amr)
{
  try { return arena_bytes_impl(cfg, amr); } catch (...) { return 0; }
}

int emma_rt_init(emma_rt** out, const emma_rt_config* cfg, const emma_rt_amr* amr, const emma_rt_fields* fields,
                 void* arena_dev, size_t arena_bytes)
{
  // *out is set as soon as the handle exists, so a failure (also an exception) leaves a handle whose message can be read
  if (out) *out = nullptr;
  try {
    return init_impl(out, cfg, amr, fields, arena_dev, arena_bytes);
  } catch (const std::bad_alloc&) {
    return fail(out ? *out : nullptr, EMMA_RT_ENOMEM, "out of host memory");
  } catch (...) {
    return fail(out ? *out : nullptr, EMMA_RT_EINVAL, "internal error (exception)");
  }
}

int emma_rt_set_sources(emma_rt* h, int64_t n_src, const double* pos_box, const double* Q)
{
  return guarded(h, true, [&] { return set_sources_impl(h, n_src, pos_box, Q); });
}

int emma_rt_step(emma_rt* h, double dt, int32_t n_steps, emma_rt_diag* diag_last)
{
  return guarded(h, true, [&] { return step_impl(h, dt, n_steps, diag_last); });
}

int emma_rt_step_host(emma_rt* h, double dt, const emma_rt_host_state* in, const emma_rt_host_state* out, emma_rt_diag* diag_last)
{
  return guarded(h, true, [&] { return step_host_impl(h, dt, in, out, diag_last); });
}

int emma_rt_read(emma_rt* h, int32_t field, int32_t level, int32_t group, void* dst, size_t bytes, int32_t dst_is_device)
{
  return guarded(h, true, [&] { return read_impl(h, field, level, group, dst, bytes, dst_is_device); });
}

int emma_rt_write(emma_rt* h, int32_t field, int32_t level, int32_t group, const void* src, size_t bytes, int32_t src_is_device)
{
  return guarded(h, true, [&] { return write_impl(h, field, level, group, src, bytes, src_is_device); });
}

int emma_rt_profile(emma_rt* h, int32_t enable, double* ms_out, int64_t* launches_out)
{
  return guarded(h, true, [&] { return profile_impl(h, enable, ms_out, launches_out); });
}

double emma_rt_dt_cfl(const emma_rt* h, double courant)
{
  return h ? courant * h->dx / (3.0 * h->cfg.c_red_cm_s) : 0.0;
}

int64_t emma_rt_level_cells(const emma_rt* h, int32_t level)
{
  if (!h || level < 0 || level > h->sh.nl) return -1;
  return h->sh.ncell[level];
}

int64_t emma_rt_kernel_launches(const emma_rt* h) { return h ? h->launches : 0; }

int emma_rt_set_schedule(emma_rt* h, int32_t fused)
{
  if (!h) return EMMA_RT_EINVAL;
  if (fused != 0 && fused != 1) return fail(h, EMMA_RT_EINVAL, "fused must be 0 or 1");
  h->fused = fused;
  return EMMA_RT_OK;
}

int emma_rt_set_inflow(emma_rt* h, int32_t face, int32_t group, const double U[4])
{
  if (!h || !U) return EMMA_RT_EINVAL;
  if (face < 0 || face > 5 || group < 0 || group >= h->sh.G) return fail(h, EMMA_RT_EINVAL, "face in 0..5, group in range");
  if (h->cfg.bc[face] != EMMA_RT_BC_INFLOW) return fail(h, EMMA_RT_EINVAL, "face %d is not an inflow face", (int)face);
  const double c = h->cfg.c_red_cm_s;
  for (int q = 0; q < 4; q++) if (!std::isfinite(U[q])) return fail(h, EMMA_RT_EINVAL, "non-finite inflow state");
  h->inflow[face][group] = make_float4((float)U[0], (float)(U[1] / c), (float)(U[2] / c), (float)(U[3] / c));
  return EMMA_RT_OK;
}

int emma_rt_set_flux(emma_rt* h, int32_t flux)
{
  if (!h) return EMMA_RT_EINVAL;
  if (flux != EMMA_RT_FLUX_GLF && flux != EMMA_RT_FLUX_HLL) return fail(h, EMMA_RT_EINVAL, "unknown flux %d", (int)flux);
  h->flux = flux;
  return EMMA_RT_OK;
}

const char* emma_rt_last_error(const emma_rt* h) { return h ? h->err : ""; }

void emma_rt_free(emma_rt* h)
{
  if (!h) return;
  if (h->diag_pinned) cudaFreeHost(h->diag_pinned);
  for (cudaEvent_t e : h->ev_in) cudaEventDestroy(e);
  for (cudaEvent_t e : h->ev_c) cudaEventDestroy(e);
  if (h->ev_start) cudaEventDestroy(h->ev_start);
  if (h->s_in) cudaStreamDestroy(h->s_in);
  if (h->s_out) cudaStreamDestroy(h->s_out);
  for (cudaEvent_t e : h->prof.pool) cudaEventDestroy(e);
  delete h;
}

}  // extern "C"
