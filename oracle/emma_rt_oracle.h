/* emma_rt_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the radiative-transfer + thermo-chemistry path of
 * arXiv 1508.07888 (EMMA), written from PAPER.md with the readings A1..A17 of DESIGN.md.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code with paper_1508_07888_b200/ (the CUDA path) and neither includes
 * the other.
 *
 * Pins: every function has one.  The two literature formulas the paper cites without printing
 * -- chi(f) between its printed limits (Levermore via PAPER.md:197) and the atomic rates / cooling
 * functions -- are pinned against other sources in tests/test_oracle_literature.py (boosted isotropic
 * field; Osterbrock & Ferland tables, Voronov 1997, Cen 1992 / Theuns et al. 1998, Rybicki & Lightman), as is the
 * H I cross-section of the group constants (exact hydrogenic closed form).  No function is "parity unpinned".
 */
#ifndef EMMA_RT_ORACLE_H
#define EMMA_RT_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_MAX_GROUPS 4
enum { ORC_OK = 0, ORC_EINVAL = -1, ORC_ENOMEM = -2, ORC_ENONFINITE = -4, ORC_ECFL = -6, ORC_ESUBCYCLE = -7 };
enum { ORC_BC_PERIODIC = 0, ORC_BC_TRANSMISSIVE = 1, ORC_BC_REFLECTIVE = 2,
       ORC_BC_INFLOW = 3 };   /* A20: ghost = a prescribed state (the plane-parallel flux of PAPER.md:562 entering a face) */
enum { ORC_F_U = 0, ORC_F_N = 1, ORC_F_F = 2, ORC_F_X = 3, ORC_F_T = 4, ORC_F_E = 5, ORC_F_N0 = 6,
       ORC_F_SUBCYCLES = 7, ORC_F_XNEUTRAL = 8 };
enum { ORC_FLUX_GLF = 0, ORC_FLUX_HLL = 1 };        /* Eq. 32 / reading A19 */
#define ORC_MAX_SUBSTEPS 65535       /* accepted sub-steps per cell per step before ORC_ESUBCYCLE */

/* physics parameters of the chemistry */
typedef struct {
  int    G;                          /* groups                                            */
  int    otsa;                       /* 1: alpha_A := alpha_B              */
  int    thermal;                    /* 0: isothermal test mode (T held, Eq. 46-48 skipped)*/
  double c;                          /* reduced speed of light (reading A3)               */
  double sigN[ORC_MAX_GROUPS];       /* Eq. 29                                            */
  double sigE[ORC_MAX_GROUPS];       /* Eq. 37                                            */
  double Emean[ORC_MAX_GROUPS];      /* Eq. 38 [erg]                                      */
  double e_tol;                      /* 0.1                                */
  int    max_halvings;
} orc_phys;

typedef struct {
  double photons_total, photons_injected, photons_absorbed, photons_recomb_emitted, photons_outflow;
  double dtau_min;
  int64_t subcycles_total, subcycles_max, halvings_total, n_nonfinite;
  double t_sim;
} orc_diag;

/* per-cell results of one chemistry call (sums are per unit volume: multiply by the cell volume) */
typedef struct {
  double absorbed;                   /* sum_p sum_i c sigN_i (1-x^p) n0 dtau N_i^{p+1}    */
  double injected;                   /* sum_p sum_i S_i dtau                              */
  double recomb;                     /* sum_p (alphaA-alphaB) x^p^2 n0^2 dtau             */
  double dtau_min;                   /* min_p of the first guess e^p/abs(H^p-Lambda^p)    */
  int    nsub, nhalv;                /* accepted sub-steps, rejected (halved) attempts    */
} orc_chem_out;

typedef struct orc orc;

/* --- stateless pieces (also used one cell at a time for sampled parity at full size) --------- */
double orc_chi(double f);                                            /* reading A2                */
void   orc_closure(const double U[4], double c, double P[9]);        /* Eq. 22-23, readings A1-A3 */
void   orc_rates(double T, double* alphaA, double* alphaB, double* beta,
                 double* cool_HI /* per n_e n_HI */, double* cool_HII_A, double* cool_HII_B /* per n_e n_HII */);
double orc_temperature(double e, double x, double n0);               /* reading A10               */
double orc_energy(double T, double x, double n0);
/* Eq. 30 + 32, unsplit 3-D, for one cell from its six face neighbours (ghosts already applied) */
void   orc_transport_stencil(double c, double dt, double dx, const double U0[4],
                             const double Um[3][4], const double Up[3][4], double out[4]);
/* the same with the interface flux chosen: ORC_FLUX_GLF (Eq. 32) or ORC_FLUX_HLL (reading A19) */
void   orc_transport_stencil_flux(int flux, double c, double dt, double dx, const double U0[4],
                                  const double Um[3][4], const double Up[3][4], double out[4]);
/* extreme eigenvalues of dF~_d/dU of the M1 system in direction d (reading A19) */
void   orc_m1_wavespeeds(const double U[4], double c, int d, double* lmin, double* lmax);
/* Eq. 43-48 sub-cycled over dt for one cell (reading A9).  U is [G][4], S is [G] (may be NULL). */
int    orc_chem_cell(const orc_phys* ph, double dt, double n0, double* x, double* e, double* U,
                     const double* S, orc_chem_out* out);

/* --- stateful driver with the library's shape -------------------------------------------------- */
orc* orc_create(int n, const int bc[6], int chemistry, const orc_phys* ph, double box_len,
                int n_levels, const int64_t* n_octs, const int64_t* const* parent,
                const float* const* U0, const float* const* n0, const float* const* x, const float* const* T);
int  orc_set_sources(orc*, int64_t n_src, const double* pos_box, const double* Q);
int  orc_set_inflow(orc*, int face, int group, const double U[4]);   /* ghost (N, Fx, Fy, Fz) of an INFLOW face */
int  orc_set_flux(orc*, int flux);          /* interface flux of the transport sweep; default ORC_FLUX_GLF */
/* standard (non-CRTA) AMR transport, reading A21: transport + chemistry on the leaves of every
 * level, dt_l = dt/2^l, finest first, fine fluxes deposited into coarser neighbours, linear (MinMod) ghosts at jumps.
 * EINVAL if a resolution jump across a face exceeds 1.  Refined cells start with their parent's radiation. */
int  orc_set_amr_transport(orc*, int on);
int  orc_write_U(orc*, int level, int group, const double* src);   /* [ncell_l][4]; level > 0 needs amr transport on */
int  orc_amr_ghost(orc*, int level, int group, const int v[3], int64_t coarse_cell, double out[4]);   /* test hook (A21) */
int  orc_restrict_U(orc*);                                         /* split cells := children mean, after orc_write_U */
int  orc_step(orc*, double dt, int n_steps, orc_diag* diag_last);
int  orc_read(const orc*, int field, int level, int group, double* dst, int64_t n_dst);
int64_t orc_level_cells(const orc*, int level);
int64_t orc_source_cell(const orc*, int64_t i_src, int* level);
/* engine sweep counters since creation (Fig. 6 scheduling check) */
void orc_counters(const orc*, int64_t transport_cells[8], int64_t chem_cells[8]);
int  orc_threads(void);
void orc_free(orc*);

#ifdef __cplusplus
}
#endif
#endif
