// chemistry.cu -- sub-cycled semi-implicit hydrogen thermo-chemistry.
//
// Eq. 43 (N), 44 (F), 45 (x), 46-48 (e), "in that order ... new information immediately used"
// (PAPER.md:306), chemical step dtau first guessed as e/(H - Lambda) and halved until e varies by <= 10 %
// (reading A9).  Point sources S = Q/dV enter Eq. 43 in every sub-step (A12).  CRTA
// (A14): leaves of refined cells start from the coarse N*, F*; split cells take the children mean.
//
// fp32 arithmetic, arranged so that nothing cancels:
//   * both x and y = 1-x are carried; Eq. 45 is evaluated as  y' = (y + r)/(1 + dtau G)  [its printed form] and
//     x' = (x + dtau G - r)/(1 + dtau G), r = alpha x^2 n0 dtau, G = beta x n0 + c sum sigma_i N_i'; whichever of
//     x', y' is <= 1/2 is kept and the other derived from it;
//   * energies are per hydrogen atom (eps = e/n0), so tiny n0^2 Lambda products never reach the denormal range;
//   * T-dependent rates are evaluated once per sub-step (state p) through lg2/ex2 (MUFU) and reused by its retries.
//
// Work distribution (north_star item 3): the level-0 pass `chem_main_kernel` is HBM-bound and gives every cell
// exactly one attempt with dtau = dt; cells whose first guess is shorter than dt, or whose attempt breaks the 10 %
// rule, are appended to a queue with one warp-aggregated atomic and left untouched.  `chem_tail_kernel` then runs
// persistent warps over that (compacted) queue: each lane owns one queued cell, advances it one accepted sub-step
// per loop trip and refills from the queue as soon as its cell is done, so lanes stay busy while any work is left.
#include "async_copy.cuh"
#include "chem_math.cuh"
#include "emma_rt_internal.cuh"

namespace emma {

namespace {

// ------------------------------------------------------------------------------------------------------------
// level 0, pass 1: every unrefined coarse cell gets one attempt with dtau = dt (HBM-bound).  The inputs of a chunk of 256
// cells (G float4 runs of 4 KB and the n0, xs, eps runs of 1 KB) are brought into a ring of shared-memory stages by
// cp.async.bulk copies that complete on mbarriers, NSTC-1 chunks ahead of the compute and at no register cost (a plain
// one-load-per-thread version kept ~60 B per thread in flight and waited on long-scoreboard stalls,
// profiles/r1b_summary.md: 14 of 18.5 cycles per issue).
// ------------------------------------------------------------------------------------------------------------
constexpr int CH = 256;                                               // cells per chunk = threads per CTA
constexpr int NSTC = 4;                                               // stages of the ring
template <int G> constexpr int chem_stage_bytes() { return CH * 16 * G + CH * 4 * 3; }
template <int G> constexpr int chem_smem_bytes() { return NSTC * chem_stage_bytes<G>() + 8 * NSTC; }

using namespace acp;

template <int G>
__global__ void __launch_bounds__(CH)
chem_main_bulk_kernel(const ChemParams cp, const LevelDev L, float4* __restrict__ U, long long ncell,
                      int* __restrict__ queue, unsigned int* __restrict__ qcount, Partial* __restrict__ parts)
{
  extern __shared__ __align__(128) unsigned char smem[];
  constexpr int SB = chem_stage_bytes<G>();
  const unsigned stage0 = (unsigned)__cvta_generic_to_shared(smem);
  const unsigned bar0 = stage0 + NSTC * SB;
  const int t = threadIdx.x, lane = t & 31;
  const long long nchunks = (ncell + CH - 1) / CH;

  // chunk i of this CTA -> stage s (arrays are 256-byte padded in the arena, so a ragged last run may be rounded
  // up to the 16-byte granularity of the copy)
  auto issue = [&](long long i, int s) {
    const long long chunk = blockIdx.x + i * gridDim.x;
    if (chunk >= nchunks) return;
    const long long base = chunk * CH;
    const unsigned cnt = (unsigned)min((long long)CH, ncell - base);
    const unsigned bU = cnt * 16u, bF = (cnt * 4u + 15u) & ~15u;
    const unsigned dst = stage0 + s * SB, bar = bar0 + 8 * s;
    mbar_expect_tx(bar, G * bU + 3 * bF);
#pragma unroll
    for (int g = 0; g < G; g++) bulk_load(dst + g * CH * 16, U + (size_t)g * ncell + base, bU, bar);
    bulk_load(dst + G * CH * 16, L.n0 + base, bF, bar);
    bulk_load(dst + G * CH * 16 + CH * 4, L.xs + base, bF, bar);
    bulk_load(dst + G * CH * 16 + CH * 8, L.eps + base, bF, bar);
  };
  if (t == 0) {
    for (int s = 0; s < NSTC; s++) mbar_init(bar0 + 8 * s, 1);
    mbar_fence_init();
  }
  __syncthreads();
  if (t == 0)
    for (int s = 0; s < NSTC; s++) issue(s, s);

  Acc acc;
  int s = 0;
  unsigned par = 0;
  for (long long i = 0;; i++) {
    const long long chunk = blockIdx.x + i * gridDim.x;
    if (chunk >= nchunks) break;
    const long long cell = chunk * CH + t;
    bool valid = cell < ncell;
    if (valid && L.refined) valid = !((L.refined[cell >> 5] >> (cell & 31)) & 1u);   // split cells: CRTA kernels
    mbar_wait(bar0 + 8 * s, par);
    CellState<G> c;
    {
      const unsigned char* st = smem + s * SB;
#pragma unroll
      for (int g = 0; g < G; g++) {
        const float4 u = *(const float4*)(st + g * CH * 16 + t * 16);
        c.N[g] = u.x; c.px[g] = u.y; c.py[g] = u.z; c.pz[g] = u.w;
      }
      c.n0 = *(const float*)(st + G * CH * 16 + t * 4);
      decode_x(*(const float*)(st + G * CH * 16 + CH * 4 + t * 4), c.x, c.y);
      c.eps = *(const float*)(st + G * CH * 16 + CH * 8 + t * 4);
    }
    __syncthreads();                                                  // every thread has taken its cell: refill
    if (t == 0) issue(i + NSTC, s);
    if (++s == NSTC) { s = 0; par ^= 1u; }
    bool defer = false;
    if (valid) {
      load_sources<G>(L, cell, c.S);
      CellTally tl;
      float dmin = FINF;
      // fast path == the first trip of the sub-cycle loop when it covers the whole step
      const float T = c.eps * frcp(KB15 * (1.f + c.x));
      const Rates r = rates_at(T, cp.otsa, c.x, c.n0);
      bool go = true;
      if (cp.thermal) {
        float hsum = 0.f;
#pragma unroll
        for (int g = 0; g < G; g++) hsum = fmaf(cp.csigE[g], c.N[g], hsum);
        const float d = c.y * hsum - c.n0 * c.x * fmaf(c.y, r.cHI, c.x * r.cHII);
        const float guess = first_guess(c.eps, d, cp.dt);
        go = guess >= cp.dt;
        if (go) dmin = guess;
      }
      float N1[G], iden[G], x1, y1, eps1;
      if (go) go = attempt<G>(cp, c, r, cp.dt, N1, iden, x1, y1, eps1);
      if (go) {
        const float k = c.y * c.n0 * cp.dt;
#pragma unroll
        for (int g = 0; g < G; g++) {
          tl.absorbed = fmaf(cp.csig[g] * k, N1[g], tl.absorbed);
          tl.injected = fmaf(c.S[g], cp.dt, tl.injected);
          c.N[g] = N1[g];
          c.px[g] = decay(c.px[g], iden[g]); c.py[g] = decay(c.py[g], iden[g]); c.pz[g] = decay(c.pz[g], iden[g]);
        }
        tl.recomb = r.rec * cp.dt;
        c.x = x1; c.y = y1; c.eps = eps1;
        tl.nsub = 1;
        store_cell<G>(L, cell, U, ncell, c, tl, cp.record);
        fold(acc, tl, c.N, G, L.dV, L.dV_total);
        acc.dtau_min = fminf(acc.dtau_min, dmin);
        if (!finite_cell<G>(c)) acc.nonfinite++;
      } else {
        defer = true;
      }
    }
    // warp-aggregated append of the deferred cells (north_star item 3: warp-level work compaction)
    const unsigned m = __ballot_sync(0xffffffffu, defer);
    if (m) {
      const int leader = __ffs(m) - 1;
      unsigned b = 0;
      if (lane == leader) b = atomicAdd(qcount, (unsigned)__popc(m));
      b = __shfl_sync(0xffffffffu, b, leader);
      if (defer) {
        queue[b + __popc(m & ((1u << lane) - 1u))] = (int)cell;
        acc.ndefer++;
      }
    }
  }
  block_reduce_store(acc, parts + blockIdx.x);
}

// ------------------------------------------------------------------------------------------------------------
// level 0, pass 2: persistent warps over the compacted queue of cells that need real sub-cycling
// ------------------------------------------------------------------------------------------------------------
template <int G>
__global__ void __launch_bounds__(128)
chem_tail_kernel(const ChemParams cp, const LevelDev L, float4* __restrict__ U, long long ncell,
                 const int* __restrict__ queue, const unsigned int* __restrict__ qcount,
                 unsigned int* __restrict__ qhead, Partial* __restrict__ parts)
{
  Acc acc;
  const unsigned nq = *qcount;
  const int lane = threadIdx.x & 31;
  CellState<G> c;
  CellTally tl;
  float rem = 0.f, dmin = FINF;
  long long cell = -1;
  bool has = false, exhausted = false;
  for (;;) {
    // refill idle lanes
    const unsigned want = __ballot_sync(0xffffffffu, !has && !exhausted);
    if (want) {
      const int leader = __ffs(want) - 1;
      unsigned b = 0;
      if (lane == leader) b = atomicAdd(qhead, (unsigned)__popc(want));
      b = __shfl_sync(0xffffffffu, b, leader);
      if (!has && !exhausted) {
        const unsigned idx = b + __popc(want & ((1u << lane) - 1u));
        if (idx < nq) {
          cell = queue[idx];
          load_cell<G>(L, cell, U, ncell, cell, c);
          tl = CellTally();
          rem = cp.dt; dmin = FINF;
          has = true;
        } else {
          exhausted = true;
        }
      }
    }
    if (!__any_sync(0xffffffffu, has)) break;
    if (has) {
      const bool ok = substep<G>(cp, c, rem, tl, dmin);
      if (!ok) acc.err |= 1u;
      if (!ok || rem <= 0.f) {
        store_cell<G>(L, cell, U, ncell, c, tl, cp.record);
        fold(acc, tl, c.N, G, L.dV, L.dV_total);
        acc.dtau_min = fminf(acc.dtau_min, dmin);
        if (!finite_cell<G>(c)) acc.nonfinite++;
        has = false;
      }
    }
  }
  block_reduce_store(acc, parts + blockIdx.x);
}

// ------------------------------------------------------------------------------------------------------------
// refined level l >= 1 (CRTA): inject -> leaf chemistry -> restriction to the parent, one thread per cell,
// 8 consecutive lanes = one oct.  Deepest level first; level 1 writes the coarse cell in place.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ float oct_sum(float v)
{
  // pairwise along x, then y, then z: (((c0+c1)+(c2+c3))+((c4+c5)+(c6+c7)))   (A14)
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  v += __shfl_xor_sync(0xffffffffu, v, 4);
  return v;
}

// Deferred octs of a refined level (row a-5; SURVEY.md section 7 hard part 6: the dense, source-hosting leaves need 10-60
// evaluations of Eq. 43-48 while their warp-mates need one).  A leaf whose single fast-path attempt does not finish the
// step makes its OCT deferred: the oct takes a slot, its finished members park their final radiation in the slot's side
// buffer, its unfinished members go to the compacted leaf queue of chem_crta_tail_kernel (one lane per leaf, refilled as
// soon as a leaf is done), and crta_restrict_kernel averages the slot afterwards.  Leaves keep no radiation between steps
// (A14), so the side buffer is the only per-leaf radiation there is; it has a slot for every oct of the level (16 G bytes
// per refined cell: 0.6 GB at config 4), so every leaf takes the same path in every run -- fast path here or tail there --
// whatever order the slots are handed out in.  No atomics on data, fixed summation order: bit-reproducible.
template <int G>
__device__ __forceinline__ void oct_restrict_store(const CellState<G>& c, float e_den, bool leader, const LevelDev& L,
                                                   const LevelDev& Lbelow, long long oct, float4* __restrict__ U0,
                                                   long long ncell0, int level)
{
  // restriction: mean of the 8 children (A14)
  float4 m[G];
#pragma unroll
  for (int g = 0; g < G; g++) {
    m[g].x = 0.125f * oct_sum(c.N[g]); m[g].y = 0.125f * oct_sum(c.px[g]);
    m[g].z = 0.125f * oct_sum(c.py[g]); m[g].w = 0.125f * oct_sum(c.pz[g]);
  }
  const float xm = 0.125f * oct_sum(c.x), ym = 0.125f * oct_sum(c.y), em = 0.125f * oct_sum(e_den);
  if (leader) {
    const long long pc = L.parent[oct];                               // split cell on the level below
    if (level == 1) {
#pragma unroll
      for (int g = 0; g < G; g++) U0[(size_t)g * ncell0 + pc] = m[g];
    } else {
#pragma unroll
      for (int g = 0; g < G; g++) L.Ut[(size_t)g * L.nocts + oct] = m[g];
    }
    Lbelow.xs[pc] = encode_x(xm, ym);
    Lbelow.eps[pc] = em / Lbelow.n0[pc];
  }
}

template <int G>
__global__ void __launch_bounds__(128, 8)
chem_refined_kernel(const ChemParams cp, const LevelDev L, const LevelDev Lbelow, const float4* __restrict__ Ut_above,
                    long long nocts_above, float4* __restrict__ U0, long long ncell0, int level, const CrtaQueue q,
                    Partial* __restrict__ parts)
{
  Acc acc;
  const long long ncell = L.ncell;                                    // multiple of 8
  const int lane = threadIdx.x & 31;
  const unsigned oct_mask = 0xffu << (lane & 24);                     // the 8 lanes of my oct
  for (long long base = (long long)blockIdx.x * blockDim.x; base < ncell; base += (long long)gridDim.x * blockDim.x) {
    const long long cell = base + threadIdx.x;
    const bool valid = cell < ncell;                                  // uniform per 8-lane group
    CellState<G> c;
    CellTally tl;
    float rem = 0.f, dmin = FINF;
    bool leaf = false;
#pragma unroll
    for (int g = 0; g < G; g++) { c.N[g] = c.px[g] = c.py[g] = c.pz[g] = 0.f; }
    c.x = c.y = c.eps = c.n0 = 0.f;
    long long oct = 0;
    if (valid) {
      oct = cell >> 3;
      const int ch = L.child ? L.child[cell] : -1;
      if (ch < 0) {
        // leaf: starts from the coarse ancestor's post-transport radiation (piecewise-constant injection); the first
        // trip of the sub-cycle loop when it covers the whole step (as chem_main_bulk_kernel)
        leaf = true;
        load_cell<G>(L, cell, U0, ncell0, (long long)L.anc0[oct], c);
        rem = cp.dt;
        const float T = c.eps * frcp(KB15 * (1.f + c.x));
        const Rates r = rates_at(T, cp.otsa, c.x, c.n0);
        bool go = true;
        if (cp.thermal) {
          float hsum = 0.f;
#pragma unroll
          for (int g = 0; g < G; g++) hsum = fmaf(cp.csigE[g], c.N[g], hsum);
          const float d = c.y * hsum - c.n0 * c.x * fmaf(c.y, r.cHI, c.x * r.cHII);
          const float guess = first_guess(c.eps, d, cp.dt);
          go = guess >= cp.dt;
          if (go) dmin = guess;
        }
        float N1[G], iden[G], x1, y1, eps1;
        if (go) go = attempt<G>(cp, c, r, cp.dt, N1, iden, x1, y1, eps1);
        if (go) {
          const float k = c.y * c.n0 * cp.dt;
#pragma unroll
          for (int g = 0; g < G; g++) {
            tl.absorbed = fmaf(cp.csig[g] * k, N1[g], tl.absorbed);
            tl.injected = fmaf(c.S[g], cp.dt, tl.injected);
            c.N[g] = N1[g];
            c.px[g] = decay(c.px[g], iden[g]); c.py[g] = decay(c.py[g], iden[g]); c.pz[g] = decay(c.pz[g], iden[g]);
          }
          tl.recomb = r.rec * cp.dt;
          c.x = x1; c.y = y1; c.eps = eps1;
          tl.nsub = 1;
          rem = 0.f;
        }
      } else {
        // split cell: restricted values were written by the kernels of the level above
#pragma unroll
        for (int g = 0; g < G; g++) {
          const float4 u = Ut_above[(size_t)g * nocts_above + ch];
          c.N[g] = u.x; c.px[g] = u.y; c.py[g] = u.z; c.pz[g] = u.w;
        }
        c.n0 = L.n0[cell]; c.eps = L.eps[cell];
        decode_x(L.xs[cell], c.x, c.y);
        if (cp.record) L.subc[cell] = 0;
      }
    }
    // ---- octs with an unfinished leaf: take a slot of the side buffer (one atomic per such oct)
    const bool unfinished = leaf && rem > 0.f;
    const unsigned um = __ballot_sync(0xffffffffu, unfinished);
    int slot = -1;
    if (um) {
      const bool oct_defers = (um & oct_mask) != 0u;
      if (oct_defers && (lane & 7) == 0) slot = (int)atomicAdd(q.counters + 2, 1u);
      slot = __shfl_sync(0xffffffffu, slot, lane & 24);              // < q.cap: there is a slot for every oct
      if (oct_defers && (lane & 7) == 0) q.oct_list[slot] = (int)oct;
      // unfinished leaves of deferred octs -> the compacted leaf queue (one warp-aggregated atomic)
      const bool enq = unfinished && slot >= 0;
      const unsigned em = __ballot_sync(0xffffffffu, enq);
      if (em) {
        const int leader = __ffs(em) - 1;
        unsigned b = 0;
        if (lane == leader) b = atomicAdd(q.counters, (unsigned)__popc(em));
        b = __shfl_sync(0xffffffffu, b, leader);
        if (enq) {
          q.lqueue[b + __popc(em & ((1u << lane) - 1u))] = slot * 8 + (int)(cell & 7);
          acc.ndefer++;
        }
      }
    }
    const bool deferred_oct = slot >= 0;
    if (leaf && rem <= 0.f) {                                         // this leaf is finished (here)
      L.xs[cell] = encode_x(c.x, c.y);
      L.eps[cell] = c.eps;
      if (cp.record) L.subc[cell] = min(tl.nsub, 65535u) | (min(tl.nhalv, 65535u) << 16);
      fold(acc, tl, c.N, G, L.dV, L.dV_total);
      acc.dtau_min = fminf(acc.dtau_min, dmin);
      if (!finite_cell<G>(c)) acc.nonfinite++;
    }
    if (deferred_oct && valid && !(leaf && rem > 0.f)) {              // finished member of a deferred oct: park its radiation
#pragma unroll
      for (int g = 0; g < G; g++)
        q.side[(size_t)g * q.cap * 8 + (size_t)slot * 8 + (cell & 7)] = make_float4(c.N[g], c.px[g], c.py[g], c.pz[g]);
    }
    oct_restrict_store<G>(c, c.eps * c.n0, valid && (cell & 7) == 0 && !deferred_oct, L, Lbelow, oct, U0, ncell0, level);
  }
  block_reduce_store(acc, parts + blockIdx.x);
}

// persistent warps over the compacted queue of unfinished refined leaves (the refined-level twin of chem_tail_kernel):
// each lane owns one leaf, advances it one accepted sub-step per trip, refills when done
template <int G>
__global__ void __launch_bounds__(128)
chem_crta_tail_kernel(const ChemParams cp, const LevelDev L, const float4* __restrict__ U0, long long ncell0,
                      const CrtaQueue q, Partial* __restrict__ parts)
{
  Acc acc;
  const unsigned nq = q.counters[0];
  const int lane = threadIdx.x & 31;
  CellState<G> c;
  CellTally tl;
  float rem = 0.f, dmin = FINF;
  long long cell = -1;
  int entry = 0;
  bool has = false, exhausted = false;
  for (;;) {
    const unsigned want = __ballot_sync(0xffffffffu, !has && !exhausted);
    if (want) {
      const int leader = __ffs(want) - 1;
      unsigned b = 0;
      if (lane == leader) b = atomicAdd(q.counters + 1, (unsigned)__popc(want));
      b = __shfl_sync(0xffffffffu, b, leader);
      if (!has && !exhausted) {
        const unsigned idx = b + __popc(want & ((1u << lane) - 1u));
        if (idx < nq) {
          entry = q.lqueue[idx];
          cell = (long long)q.oct_list[entry >> 3] * 8 + (entry & 7);
          load_cell<G>(L, cell, U0, ncell0, (long long)L.anc0[cell >> 3], c);
          tl = CellTally();
          rem = cp.dt; dmin = FINF;
          has = true;
        } else {
          exhausted = true;
        }
      }
    }
    if (!__any_sync(0xffffffffu, has)) break;
    if (has) {
      const bool ok = substep<G>(cp, c, rem, tl, dmin);
      if (!ok) acc.err |= 1u;
      if (!ok || rem <= 0.f) {
        L.xs[cell] = encode_x(c.x, c.y);
        L.eps[cell] = c.eps;
        if (cp.record) L.subc[cell] = min(tl.nsub, 65535u) | (min(tl.nhalv, 65535u) << 16);
#pragma unroll
        for (int g = 0; g < G; g++) q.side[(size_t)g * q.cap * 8 + entry] = make_float4(c.N[g], c.px[g], c.py[g], c.pz[g]);
        fold(acc, tl, c.N, G, L.dV, L.dV_total);
        acc.dtau_min = fminf(acc.dtau_min, dmin);
        if (!finite_cell<G>(c)) acc.nonfinite++;
        has = false;
      }
    }
  }
  block_reduce_store(acc, parts + blockIdx.x);
}

// children mean of the deferred octs, after the tail: 8 lanes per slot
template <int G>
__global__ void __launch_bounds__(128)
crta_restrict_kernel(const LevelDev L, const LevelDev Lbelow, float4* __restrict__ U0, long long ncell0, int level,
                     const CrtaQueue q)
{
  const long long total = 8LL * min(q.counters[2], (unsigned)q.cap);
  const int lane = threadIdx.x & 31;
  for (long long base = (long long)blockIdx.x * blockDim.x + (threadIdx.x - lane); base < total; base += (long long)gridDim.x * blockDim.x) {
    const long long i = base + lane;                                  // warp-uniform trip count: the shuffles below are safe
    const bool valid = i < total;
    CellState<G> c;
#pragma unroll
    for (int g = 0; g < G; g++) { c.N[g] = c.px[g] = c.py[g] = c.pz[g] = 0.f; }
    c.x = c.y = c.eps = c.n0 = 0.f;
    long long oct = 0;
    if (valid) {
      oct = q.oct_list[i >> 3];
      const long long cell = oct * 8 + (i & 7);
#pragma unroll
      for (int g = 0; g < G; g++) {
        const float4 u = q.side[(size_t)g * q.cap * 8 + i];
        c.N[g] = u.x; c.px[g] = u.y; c.py[g] = u.z; c.pz[g] = u.w;
      }
      c.n0 = L.n0[cell]; c.eps = L.eps[cell];
      decode_x(L.xs[cell], c.x, c.y);
    }
    oct_restrict_store<G>(c, c.eps * c.n0, valid && (i & 7) == 0, L, Lbelow, oct, U0, ncell0, level);
  }
}

// chemistry off: Eq. 43 degenerates to N += S dt in the source cells (A9); sources are folded to the coarse level
template <int G>
__global__ void inject_kernel(const LevelDev L, float dt, float4* __restrict__ U, long long ncell, Partial* parts)
{
  Acc acc;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < L.n_src; i += gridDim.x * blockDim.x) {
    const long long cell = L.src_cell[i];
#pragma unroll
    for (int g = 0; g < G; g++) {
      const float add = L.src_S[(size_t)i * G + g] * dt;
      U[(size_t)g * ncell + cell].x += add;
      acc.injected += (double)add * L.dV;
      acc.total += (double)add * L.dV;
    }
  }
  block_reduce_store(acc, parts + blockIdx.x);
}

// children mean of n0, x, e at init (bottom-up), 8 lanes per oct
__global__ void restrict_init_kernel(const LevelDev L, const LevelDev Lbelow)
{
  const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = cell < L.ncell;
  float n0 = 0.f, x = 0.f, y = 0.f, e = 0.f;
  if (valid) {
    n0 = L.n0[cell];
    decode_x(L.xs[cell], x, y);
    e = L.eps[cell] * n0;
  }
  const float nm = 0.125f * oct_sum(n0), xm = 0.125f * oct_sum(x), ym = 0.125f * oct_sum(y), em = 0.125f * oct_sum(e);
  if (valid && (cell & 7) == 0) {
    const long long pc = L.parent[cell >> 3];
    Lbelow.n0[pc] = nm;
    Lbelow.xs[pc] = encode_x(xm, ym);
    Lbelow.eps[pc] = em / nm;
  }
}

template <int G>
int chem_tail_G(const ChemParams& cp, const LevelDev& L0, float4* U, long long ncell, int* queue, unsigned int* qcount,
                Partial* parts, int* n_parts, int sm_count, cudaStream_t st, Profiler* pf)
{
  int nt = sm_count * 8;
  if (nt > MAX_PART_BLOCKS) nt = MAX_PART_BLOCKS;
  pf->begin(EMMA_RT_K_CHEM_TAIL);
  chem_tail_kernel<G><<<nt, 128, 0, st>>>(cp, L0, U, ncell, queue, qcount, qcount + 1, parts);
  pf->end();
  *n_parts = nt;
  return 1;
}

template <int G>
int chem_level0_G(const ChemParams& cp, const LevelDev& L0, float4* U, long long ncell, int* queue, unsigned int* qcount,
                  Partial* parts, int* n_parts, int sm_count, int ctas_per_sm, cudaStream_t st, Profiler* pf)
{
  const long long want = (ncell + CH - 1) / CH;
  long long cap = (long long)sm_count * (ctas_per_sm > 0 ? ctas_per_sm : 1);      // persistent CTAs: as many as fit per SM
  if (cap > MAX_PART_BLOCKS) cap = MAX_PART_BLOCKS;
  const int nb = (int)(want < cap ? want : cap);
  pf->begin(EMMA_RT_K_CHEM_MAIN);
  chem_main_bulk_kernel<G><<<nb, CH, chem_smem_bytes<G>(), st>>>(cp, L0, U, ncell, queue, qcount, parts);
  pf->end();
  *n_parts = nb;
  if (!cp.thermal) return 1;                                          // isothermal mode never defers
  int nt = 0;
  chem_tail_G<G>(cp, L0, U, ncell, queue, qcount, parts + nb, &nt, sm_count, st, pf);
  *n_parts = nb + nt;
  return 2;
}

template <int G>
cudaError_t chem_configure_G(int* occ)
{
  cudaError_t e = cudaFuncSetAttribute(chem_main_bulk_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, chem_smem_bytes<G>());
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, chem_main_bulk_kernel<G>, CH, chem_smem_bytes<G>());
}

}  // namespace

// Per-device set-up of the chemistry kernels for G groups (called by emma_rt_init with the handle's device current):
// opts the bulk main pass into its dynamic shared memory and returns how many of its CTAs fit on an SM.
cudaError_t configure_chemistry(int G, int* ctas_per_sm)
{
  switch (G) {
    case 1: return chem_configure_G<1>(ctas_per_sm);
    case 2: return chem_configure_G<2>(ctas_per_sm);
    case 3: return chem_configure_G<3>(ctas_per_sm);
    default: return chem_configure_G<4>(ctas_per_sm);
  }
}

int launch_chem_level0(const ChemParams& cp, const LevelDev& L0, float4* U, long long ncell, int* queue,
                       unsigned int* qcount, Partial* parts, int* n_parts, int sm_count, int ctas_per_sm, cudaStream_t st,
                       Profiler* pf)
{
  switch (cp.G) {
    case 1: return chem_level0_G<1>(cp, L0, U, ncell, queue, qcount, parts, n_parts, sm_count, ctas_per_sm, st, pf);
    case 2: return chem_level0_G<2>(cp, L0, U, ncell, queue, qcount, parts, n_parts, sm_count, ctas_per_sm, st, pf);
    case 3: return chem_level0_G<3>(cp, L0, U, ncell, queue, qcount, parts, n_parts, sm_count, ctas_per_sm, st, pf);
    default: return chem_level0_G<4>(cp, L0, U, ncell, queue, qcount, parts, n_parts, sm_count, ctas_per_sm, st, pf);
  }
}

// the compacted tail alone (after the fused pass, which fills the queue itself)
int launch_chem_tail(const ChemParams& cp, const LevelDev& L0, float4* U, long long ncell, int* queue,
                     unsigned int* qcount, Partial* parts, int* n_parts, int sm_count, cudaStream_t st, Profiler* pf)
{
  *n_parts = 0;
  if (!cp.thermal) return 0;                                          // isothermal mode never defers
  switch (cp.G) {
    case 1: return chem_tail_G<1>(cp, L0, U, ncell, queue, qcount, parts, n_parts, sm_count, st, pf);
    case 2: return chem_tail_G<2>(cp, L0, U, ncell, queue, qcount, parts, n_parts, sm_count, st, pf);
    case 3: return chem_tail_G<3>(cp, L0, U, ncell, queue, qcount, parts, n_parts, sm_count, st, pf);
    default: return chem_tail_G<4>(cp, L0, U, ncell, queue, qcount, parts, n_parts, sm_count, st, pf);
  }
}

int launch_chem_refined(const ChemParams& cp, const LevelDev* lv, int level, int n_levels, float4* U, long long ncell0,
                        const CrtaQueue& q, Partial* parts, int* n_parts, int sm_count, cudaStream_t st)
{
  const LevelDev& L = lv[level];
  if (L.ncell == 0) { *n_parts = 0; return 0; }
  long long want = (L.ncell + 127) / 128;
  // persistent grid: whole waves of 8 CTAs per SM
  const long long cap = (sm_count > 0 && (long long)sm_count * 8 <= MAX_PART_BLOCKS) ? (long long)sm_count * 8 : MAX_PART_BLOCKS;
  const int nb = (int)(want < cap ? want : cap);
  const float4* Ut_above = (level < n_levels) ? lv[level + 1].Ut : nullptr;
  const long long nocts_above = (level < n_levels) ? lv[level + 1].nocts : 0;
  const bool tail = cp.thermal && q.cap > 0;                          // isothermal mode never leaves a leaf unfinished
  int nt = 0;
  if (tail) {
    nt = sm_count * 8;
    if (nt > MAX_PART_BLOCKS) nt = MAX_PART_BLOCKS;
    cudaMemsetAsync(q.counters, 0, 3 * sizeof(unsigned int), st);
  }
  long long rwant = ((long long)q.cap * 8 + 127) / 128;
  const int nr = (int)(rwant < cap ? rwant : cap);
#define CRTA_LAUNCH(GG)                                                                                                       \
  chem_refined_kernel<GG><<<nb, 128, 0, st>>>(cp, L, lv[level - 1], Ut_above, nocts_above, U, ncell0, level, q, parts);          \
  if (tail) {                                                                                                                 \
    chem_crta_tail_kernel<GG><<<nt, 128, 0, st>>>(cp, L, U, ncell0, q, parts + nb);                                             \
    crta_restrict_kernel<GG><<<nr, 128, 0, st>>>(L, lv[level - 1], U, ncell0, level, q);                                        \
  }
  switch (cp.G) {
    case 1: { CRTA_LAUNCH(1) } break;
    case 2: { CRTA_LAUNCH(2) } break;
    case 3: { CRTA_LAUNCH(3) } break;
    default: { CRTA_LAUNCH(4) } break;
  }
#undef CRTA_LAUNCH
  if (tail) cudaMemsetAsync(q.counters, 0, 3 * sizeof(unsigned int), st);   // the level-0 passes share the queue and its counters
  *n_parts = nb + nt;
  return tail ? 3 : 1;
}

int launch_inject_sources(const LevelDev& L0, int G, float dt, float4* U, long long ncell0, Partial* parts, int* n_parts,
                          cudaStream_t st)
{
  if (L0.n_src == 0) { *n_parts = 0; return 0; }
  int nb = (L0.n_src + 127) / 128;
  if (nb > 64) nb = 64;
  switch (G) {
    case 1: inject_kernel<1><<<nb, 128, 0, st>>>(L0, dt, U, ncell0, parts); break;
    case 2: inject_kernel<2><<<nb, 128, 0, st>>>(L0, dt, U, ncell0, parts); break;
    case 3: inject_kernel<3><<<nb, 128, 0, st>>>(L0, dt, U, ncell0, parts); break;
    default: inject_kernel<4><<<nb, 128, 0, st>>>(L0, dt, U, ncell0, parts); break;
  }
  *n_parts = nb;
  return 1;
}

int launch_restrict_init(const LevelDev* lv, int level, cudaStream_t st)
{
  const LevelDev& L = lv[level];
  if (L.ncell == 0) return 0;
  const int nb = (int)((L.ncell + 127) / 128);
  restrict_init_kernel<<<nb, 128, 0, st>>>(L, lv[level - 1]);
  return 1;
}

}  // namespace emma
