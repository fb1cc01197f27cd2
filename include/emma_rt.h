/* emma_rt.h -- C-ABI of the B200-native radiative-transfer + thermo-chemistry hot path of EMMA
 * (arXiv 1508.07888).  Citations are /root/reference/PAPER.md line numbers; "A<n>" are the readings of the
 * paper listed in DESIGN.md section 2.1.
 *
 * What one coupled step computes:
 *   1. explicit M1 transport on the coarse level, per photon group: Levermore closure (Eq. 22-23, A1/A2),
 *      Lax-Friedrichs/GLF interface flux (Eq. 32) with the reduced speed of light (A3), unsplit
 *      conservative update (Eq. 30, A4), boundary conditions of PAPER.md:436 (A13);
 *   2. CRTA injection of the coarse radiation into refined cells (A14);
 *   3. hydrogen thermo-chemistry on every leaf cell, sub-cycled semi-implicitly (Eq. 43-48, A5-A9), with
 *      point sources entering Eq. 43 (A12);
 *   4. restriction of N, F, x, e to split cells (children mean, A14);
 *   5. fp64 diagnostics (photon budget A15, min chemical time, sub-cycle counts).
 * With config.amr_transport = 1 steps 1-4 become the standard AMR scheme (transport and chemistry on the leaves of
 * every level with dt_l = dt / 2^l; see the field's comment).
 *
 * Conventions
 *   - All pointers are HOST pointers unless the argument name ends in `_dev` or the call has an
 *     `*_is_device` flag.  Plain C types only; no C++/torch types cross this boundary.
 *   - Units are cgs: N [photons cm^-3], F [photons cm^-2 s^-1], n0 [cm^-3], T [K], e [erg cm^-3], Q [photons s^-1].
 *   - Coarse cell id = ix + n*(iy + n*iz) (x fastest).  Cell id on refined level l = oct*8 + (ix + 2*iy + 4*iz);
 *     arrays on level l have 8*n_octs[l-1] entries in oct order.  Entries of split cells are ignored on input and
 *     hold the restricted (children-mean) value on output.
 *   - Ownership: the handle owns host bookkeeping only.  Device memory is ONE caller-allocated arena
 *     (`emma_rt_arena_bytes`), which must stay alive and untouched until `emma_rt_free`.  Host input arrays are
 *     borrowed for the duration of the call.  The CUDA stream is borrowed.
 *   - Errors: every entry point returns EMMA_RT_OK or a negative code; nothing throws, aborts or prints.
 *     `emma_rt_last_error` gives a handle-owned message.  There is no CPU fallback: without a CUDA device
 *     `emma_rt_init` returns EMMA_RT_ECUDA.
 *   - Threading: one handle <-> one stream, not re-entrant.  A process may hold handles on several devices: every entry
 *     point that launches work makes the handle's device current (cudaSetDevice) and leaves it current.
 *   - Input validation: `emma_rt_init` and `emma_rt_write` with HOST buffers refuse (EMMA_RT_EINVAL) n0 <= 0, T <= 0,
 *     x outside [0, 1] and non-finite n0, x, T; a non-finite U is accepted and reported by the next step
 *     (EMMA_RT_ENONFINITE).  A refused write has still stored the field (x clamped to [0, 1]): write it again with valid
 *     values, or discard the handle after a refused init.  Device-buffer writes are stream-ordered and not validated (a
 *     NaN stays a NaN).
 *   - Environment: five tuning knobs for experiments are read ONCE, by `emma_rt_init`, and ignored when unset, not a
 *     number or out of range: EMMA_RT_TUNE_NZC (z-chunks per tile column of the dense passes, 1..n; a pass whose
 *     partial-sum slots that count would overflow keeps its own choice), EMMA_RT_TUNE_NST
 *     (stages of the transport TMA ring: 4, 6, 8), EMMA_RT_TUNE_TMA (0: non-TMA transport kernel), EMMA_RT_TUNE_FUSED
 *     (0: two-pass schedule), EMMA_RT_TUNE_CHEMCTAS (persistent CTAs per SM of the chemistry main pass, 1..32).  None
 *     changes results beyond fp32 rounding order of nothing (same arithmetic); `emma_rt_step` reads no environment.
 *   - Sync: `emma_rt_step` only enqueues work unless `diag_last != NULL` (then it waits for the stream);
 *     `emma_rt_read` / `emma_rt_write` with host buffers wait for the stream.
 */
#ifndef EMMA_RT_H
#define EMMA_RT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define EMMA_RT_API __attribute__((visibility("default")))
#else
#define EMMA_RT_API
#endif

#define EMMA_RT_ABI_VERSION 2
#define EMMA_RT_MAX_GROUPS 4
#define EMMA_RT_MAX_LEVELS 4          /* refined levels above the base */
#define EMMA_RT_MAX_SUBSTEPS 65535    /* accepted sub-steps per cell per step before EMMA_RT_ESUBCYCLE (A9) */

typedef struct emma_rt emma_rt;      /* opaque */

enum { EMMA_RT_OK = 0, EMMA_RT_EINVAL = -1, EMMA_RT_ENOMEM = -2, EMMA_RT_ECUDA = -3, EMMA_RT_ENONFINITE = -4,
       EMMA_RT_ESTATE = -5, EMMA_RT_ECFL = -6, EMMA_RT_ESUBCYCLE = -7 };

/* boundary conditions: periodic by nature; transmissive = ghost copies the cell;
 * reflective = the same with the face-normal flux component inverted (A13) */
enum { EMMA_RT_BC_PERIODIC = 0, EMMA_RT_BC_TRANSMISSIVE = 1, EMMA_RT_BC_REFLECTIVE = 2,
       EMMA_RT_BC_INFLOW = 3 };   /* ghost = a prescribed state, see emma_rt_set_inflow (reading A20) */

/* fields of emma_rt_read / emma_rt_write.  Element type and count per cell in brackets. */
enum {
  EMMA_RT_FIELD_U = 0,          /* [float x4] (N,Fx,Fy,Fz) of `group`; level 0 (any level with amr_transport; after a write
                                               split cells are re-restricted before the next step)  (read, write) */
  EMMA_RT_FIELD_N = 1,          /* [float]    photon density of `group`; level 0 (any level with amr_transport) (read)  */
  EMMA_RT_FIELD_F = 2,          /* [float x3] photon flux of `group`; level 0 (any level with amr_transport)    (read)  */
  EMMA_RT_FIELD_X = 3,          /* [float]    ionised fraction x                                (read, write) */
  EMMA_RT_FIELD_T = 4,          /* [float]    temperature, T = e / (1.5 (1+x) n0 k_B) (A10)     (read, write: uses the x
                                               currently stored, so write X before T)                          */
  EMMA_RT_FIELD_E = 5,          /* [float]    internal energy density e                         (read)        */
  EMMA_RT_FIELD_N0 = 6,         /* [float]    hydrogen number density n0                        (read, write) */
  EMMA_RT_FIELD_SUBCYCLES = 7,  /* [uint32]   last step: accepted sub-steps | rejected (halved) attempts << 16,
                                               each saturating at 65535; needs config.record_subcycles (read) */
  EMMA_RT_FIELD_XNEUTRAL = 8    /* [float]    neutral fraction 1-x, kept to full relative precision (read)     */
};

typedef struct {
  uint32_t struct_size;         /* sizeof(emma_rt_config), checked                                            */
  uint32_t abi_version;         /* EMMA_RT_ABI_VERSION                                                        */
  int32_t  n_coarse;            /* cells per side of the base level, 2^lc in the paper; >= 2    */
  int32_t  n_groups;            /* 1..EMMA_RT_MAX_GROUPS                                  */
  int32_t  bc[6];               /* -x,+x,-y,+y,-z,+z                                                          */
  int32_t  otsa;                /* 1: alpha_A := alpha_B in Eq. 33/35, no recombination radiation */
  int32_t  chemistry;           /* 0: transport + sources only (N += S dt); 1: Eq. 43-48                      */
  int32_t  thermal;             /* 0: isothermal test mode (T held, Eq. 46-48 skipped, one sub-step); 1: full */
  int32_t  record_subcycles;    /* 1: keep per-cell sub-cycle signatures of the last step (4 B/cell)          */
  int32_t  max_halvings;        /* guard on the "divide by 2" retries of one sub-step          */
  int32_t  device;              /* CUDA ordinal                                                               */
  int64_t  max_source_cells;    /* capacity of the per-level source lists (0 -> 65536)                        */
  double   box_len_cm;          /* L; dx = L / n_coarse                                                       */
  double   c_red_cm_s;          /* reduced speed of light                                      */
  double   sigma_N[EMMA_RT_MAX_GROUPS];   /* Eq. 29 [cm^2]                                                    */
  double   sigma_E[EMMA_RT_MAX_GROUPS];   /* Eq. 37 [cm^2]                                                    */
  double   E_mean[EMMA_RT_MAX_GROUPS];    /* Eq. 38 [erg]                                                     */
  double   e_tol;               /* 0.1                                                         */
  void*    stream;              /* cudaStream_t of the caller (e.g. torch's current stream); 0 = default      */
  int32_t  amr_transport;       /* 0: CRTA, transport on the coarse level only (the default).
                                   1: the standard AMR scheme (reading A21): every
                                   level carries (N, F); advance(l, dt) = advance(l+1, dt/2) twice, then Eq. 30 and
                                   Eq. 43-48 on the leaves of level l, then split cells := children mean.  Fluxes
                                   through a coarse-fine face are computed by the fine cells from a MinMod-limited
                                   linear ghost and deposited into the coarse leaf.  Needs face jumps <= 1 (else
                                   EMMA_RT_EINVAL at init), <= 3 refined levels; either interface flux
                                   (emma_rt_set_flux); U0 is injected into the refined cells at init; FIELD_U/N/F can then be read and U written on any level */
  int32_t  reserved0;
} emma_rt_config;

typedef struct {                /* static AMR description (host pointers, borrowed during init only)          */
  int32_t  n_levels;            /* refined levels above the base: 0 = uniform grid; <= EMMA_RT_MAX_LEVELS     */
  const int64_t* n_octs;        /* [n_levels]                                                                 */
  const int64_t* const* parent; /* [n_levels][n_octs[l]] -> id of the split cell on the level below           */
} emma_rt_amr;

typedef struct {                /* initial state (host pointers, borrowed during init only)                   */
  const float* const* U0;       /* [n_groups] -> n^3 x (N,Fx,Fy,Fz); NULL (or a NULL entry) => zeros          */
  const float* const* n0;       /* [n_levels+1] hydrogen number density                                       */
  const float* const* x;        /* [n_levels+1] ionised fraction in [0,1]                                     */
  const float* const* T;        /* [n_levels+1] temperature [K]; the library stores the energy (A10)          */
} emma_rt_fields;

typedef struct {                /* diagnostics of the LAST step of an emma_rt_step call (A15), plus totals     */
  double  photons_total;        /* sum over leaves of sum_g N_g dV after the step                             */
  double  photons_injected;     /* sum S_g dtau dV  (= sum Q dt)                                              */
  double  photons_absorbed;     /* sum c sigma_g (1-x^p) n0 dtau N_g^{p+1} dV, the sink of Eq. 43             */
  double  photons_recomb_emitted; /* (alpha_A-alpha_B) x^2 n0^2 dtau dV into group 1; 0 under OTSA (A6)       */
  double  photons_outflow;      /* net GLF flux through non-periodic box faces x dx^2 dt                      */
  double  dtau_min;             /* min over leaves and sub-steps of the first guess e/abs(H-Lambda) */
  int64_t subcycles_total;      /* accepted sub-steps, all leaves                                             */
  int64_t subcycles_max;        /* max accepted sub-steps of one cell                                         */
  int64_t halvings_total;       /* rejected attempts                                                          */
  int64_t n_nonfinite;          /* cells holding a non-finite N, F, x or e after the step                     */
  int64_t n_deferred;           /* leaves that needed more than the single fast-path attempt                  */
  double  t_sim;                /* simulated time since init [s]                                              */
} emma_rt_diag;

/* Bytes of device memory the arena must hold for this problem; 0 if the arguments are invalid. */
EMMA_RT_API size_t emma_rt_arena_bytes(const emma_rt_config* cfg, const emma_rt_amr* amr);

/* Validate, lay out the arena (256-byte aligned device pointer `arena_dev`, >= emma_rt_arena_bytes), upload the
 * fields, compute e from T (A10) and the restricted values of split cells.  `amr` may be NULL (uniform grid). */
EMMA_RT_API int emma_rt_init(emma_rt** out, const emma_rt_config* cfg, const emma_rt_amr* amr, const emma_rt_fields* fields,
                 void* arena_dev, size_t arena_bytes);

/* Replace the point-source list.  pos_box: [n_src][3] in [0,1)^3 box units; Q: [n_src][n_groups] photons/s (fp64:
 * Q ~ 1e48 overflows fp32).  Each source goes to the LEAF cell containing it, S_g = Q_g / dV_leaf; sources in the
 * same cell add (A12).  Invalid position / negative or non-finite Q -> EMMA_RT_EINVAL and the list is unchanged. */
EMMA_RT_API int emma_rt_set_sources(emma_rt* h, int64_t n_src, const double* pos_box, const double* Q);

/* courant * dx / (3 c_red): the largest stable step is courant = 1 (A4). */
EMMA_RT_API double emma_rt_dt_cfl(const emma_rt* h, double courant);

/* Advance n_steps coupled steps of size dt.  dt > dx/(3 c_red) -> EMMA_RT_ECFL, state untouched.
 * n_steps == 0 with diag_last != NULL: a state query (photons_total and t_sim of the current state, summed on the device).
 * diag_last == NULL: asynchronous.  Otherwise waits and fills *diag_last; returns EMMA_RT_ENONFINITE /
 * EMMA_RT_ESUBCYCLE if the last step saw them (the step still completed). */
EMMA_RT_API int emma_rt_step(emma_rt* h, double dt, int32_t n_steps, emma_rt_diag* diag_last);

/* One coupled step for a caller whose state lives in HOST memory -- the paper's own mode of operation, whose host <-> device
 * traffic took ~70 % of its GPU engines' time.  Equivalent, bit for bit, to
 *     emma_rt_write(U_g, X, T from `in`) -> emma_rt_step(h, dt, 1, diag) -> emma_rt_read(U_g, X, T into `out`),
 * but the grid goes through the device in z-slabs on three streams: the upload of slab k+1, the fused transport +
 * chemistry pass over slab k and the download of slab k-1 overlap, so both directions of the link are busy at once.
 * `in` and `out` are level-0 host arrays (U[g]: n^3 x (N,Fx,Fy,Fz) per group; x, T: n^3), pinned for the copies to be
 * asynchronous (pageable memory works, serialised); `out` may be the same arrays as `in`.  n0 and the sources stay on the
 * device.  Needs a uniform grid (n_levels = 0), chemistry = 1, the GLF flux, the fused schedule and no inflow face, else
 * EMMA_RT_ESTATE.  Waits for completion; afterwards the device holds the new state too.  Errors as emma_rt_step, plus
 * EMMA_RT_EINVAL for invalid x / T in `in` (see "Input validation"; the step has then run on the clamped values). */
typedef struct {
  float* const* U;              /* [n_groups] -> n^3 x 4 floats */
  float* x;                     /* n^3 */
  float* T;                     /* n^3 */
} emma_rt_host_state;
EMMA_RT_API int emma_rt_step_host(emma_rt* h, double dt, const emma_rt_host_state* in, const emma_rt_host_state* out,
                                  emma_rt_diag* diag_last /* nullable */);

/* Copy a field of one level (and group) out of / into the library.  dst/src holds exactly n_cells(level) elements
 * of the field's type; `bytes` must match.  *_is_device != 0: the pointer is a device pointer on the same device
 * and the copy is stream-ordered; otherwise it is a host pointer and the call waits for the stream. */
EMMA_RT_API int emma_rt_read(emma_rt* h, int32_t field, int32_t level, int32_t group, void* dst, size_t bytes, int32_t dst_is_device);
EMMA_RT_API int emma_rt_write(emma_rt* h, int32_t field, int32_t level, int32_t group, const void* src, size_t bytes, int32_t src_is_device);

EMMA_RT_API int64_t emma_rt_level_cells(const emma_rt* h, int32_t level);      /* n^3 or 8*n_octs; -1 if out of range       */
EMMA_RT_API int64_t emma_rt_kernel_launches(const emma_rt* h);                 /* kernels launched by this handle so far     */
/* Per-kernel device timing.  Waits for the stream, returns in ms_out / launches_out (each EMMA_RT_K_COUNT long,
 * nullable) the summed CUDA-event durations and launch counts of the emma_rt_step kernels recorded since the last
 * call, clears them, and switches recording on (enable != 0) or off for the steps that follow.  Off by default. */
enum { EMMA_RT_K_TRANSPORT = 0, EMMA_RT_K_CHEM_MAIN = 1, EMMA_RT_K_CHEM_TAIL = 2, EMMA_RT_K_CHEM_REFINED = 3,
       EMMA_RT_K_FINALIZE = 4, EMMA_RT_K_OTHER = 5, EMMA_RT_K_FUSED = 6,
       EMMA_RT_K_AMR_TRANSPORT = 7 /* refined-level transport + ghost faces */, EMMA_RT_K_AMR_CHEM = 8 /* refined-level chemistry */,
       EMMA_RT_K_COUNT = 9 };
EMMA_RT_API int emma_rt_profile(emma_rt* h, int32_t enable, double* ms_out, int64_t* launches_out);
/* Schedule of the coupled step on the unrefined coarse cells (same result up to fp32 rounding order of nothing: both
 * schedules run the same arithmetic).  fused = 1 (default): ONE pass does the transport update (Eq. 30, 32) and the
 * first trip of the sub-cycle loop (Eq. 43-48), so the radiation field crosses HBM once per step; fused = 0: a
 * transport pass followed by a chemistry pass.  Ignored when chemistry = 0.  Returns EMMA_RT_OK or EINVAL. */
EMMA_RT_API int emma_rt_set_schedule(emma_rt* h, int32_t fused);
/* Inflow boundary (reading A20; "the x = 0 boundary is a source of flux of the required
 * rate"): the ghost cells outside a face whose bc is EMMA_RT_BC_INFLOW hold the state U = (N, Fx, Fy, Fz) [photons cm^-3,
 * photons cm^-2 s^-1] given here for `group` (zeros until set); a plane-parallel flux F entering through -x is
 * (F / c_red, F, 0, 0).  face = 0..5 = -x,+x,-y,+y,-z,+z.  With an inflow face the step runs the two-pass schedule and the
 * non-TMA transport kernel.  The net flux through the face counts (negative) in photons_outflow.  Returns OK / EINVAL. */
EMMA_RT_API int emma_rt_set_inflow(emma_rt* h, int32_t face, int32_t group, const double U[4]);
/* Interface flux of the transport update (Eq. 30).  EMMA_RT_FLUX_GLF (default): the Lax-Friedrichs / GLF flux of Eq. 32
 * (PAPER.md:246).  EMMA_RT_FLUX_HLL: the HLL flux the paper names as its less diffusive successor (
 * DESIGN.md reading A19):  F = [l+ F~_L - l- F~_R + l+ l- (U_R - U_L)] / (l+ - l-),  l+ = max(0, lmax_L, lmax_R),
 * l- = min(0, lmin_L, lmin_R), lmin/lmax the extreme eigenvalues of the M1 flux Jacobian in the face direction.
 * With HLL the coupled step runs the two-pass schedule (the fused pass implements Eq. 32 only).  Returns OK / EINVAL. */
enum { EMMA_RT_FLUX_GLF = 0, EMMA_RT_FLUX_HLL = 1 };
EMMA_RT_API int emma_rt_set_flux(emma_rt* h, int32_t flux);
EMMA_RT_API const char* emma_rt_last_error(const emma_rt* h);                  /* handle-owned; "" if none                   */
EMMA_RT_API void emma_rt_free(emma_rt* h);                                     /* does not free the arena                    */

/* ---- the one entry point that allocates nothing ------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it)
 * and so cannot create a handle, whose arena is where every other kernel keeps its scratch.
 *
 * Photon total of A15 (emma_rt_diag.photons_total, Eq. 30 conserves it up to sources and sinks):
 *     *total_dev = dV * sum_{i < n_cellgroups} U_dev[i].N
 * -- the same kernels, grid and summation order as the state query emma_rt_step(h, dt, 0, &diag), hence the same bits.
 *   U_dev         DEVICE pointer, borrowed: n_cellgroups x (N, Fx, Fy, Fz) float, 16-byte aligned -- the layout of
 *                 EMMA_RT_FIELD_U, the groups of a level one after the other (only N is read); may be NULL if n = 0
 *   n_cellgroups  cells x groups, 0 .. EMMA_RT_NOALLOC_MAX_CELLGROUPS (2^33: the largest grid emma_rt_init accepts,
 *                 1290^3 x 4 groups, fits); beyond that EMMA_RT_EINVAL and nothing is launched: sum the array in pieces
 *   dV            cell volume [cm^3], positive and finite
 *   total_dev     DEVICE pointer to one double, written by the second kernel (stream-ordered; the call does not wait)
 *   stream        cudaStream_t of the caller, borrowed; 0 = default stream
 *   err, err_len  optional HOST buffer for the error text ("" on success); may be NULL
 * Returns EMMA_RT_OK, EMMA_RT_EINVAL (bad argument, size beyond the maximum) or EMMA_RT_ECUDA.  Calls no cudaMalloc /
 * cudaFree / allocating routine, synchronises nothing, and launches two kernels on `stream`.  The scratch (1024 block sums,
 * 88 KB) is a static device array that every GPU which loads the library holds until the process exits; its device
 * address is looked up (cudaGetSymbolAddress) in the first call on each device, with the caller's current device -- make
 * that first call (n_cellgroups = 0 will do) outside graph capture.  ALL calls share the scratch: calls on one stream are
 * safe (every slot a call reads it has written itself: nothing is carried over from the last call), calls that overlap on
 * the GPU (several streams, concurrent graph replays) race. */
#define EMMA_RT_NOALLOC_MAX_CELLGROUPS (1ll << 33)
EMMA_RT_API int emma_rt_photons_total_noalloc(const void* U_dev, int64_t n_cellgroups, double dV, double* total_dev,
                                              void* stream, char* err, size_t err_len);

#ifdef __cplusplus
}
#endif
#endif
