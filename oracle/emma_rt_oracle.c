/* emma_rt_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see emma_rt_oracle.h).
 *
 * fp64, literal, one equation at a time, in the paper's order and notation.  No blocking, no fusion:
 * face fluxes are formed explicitly (Eq. 32), the closure is recomputed wherever it is needed, Eq. 45
 * is evaluated as printed.  The only parallelism is an OpenMP `parallel for` over independent cells
 * (Jacobi transport reads the old buffer only; chemistry is cell-local), which reorders nothing
 * inside a cell; sums for the diagnostics are reduced per z-slab / per oct block and then added
 * serially in index order so results do not depend on the thread count.
 *
 * Citations are PAPER.md line numbers; "A<n>" are the readings listed in DESIGN.md.
 */
#include "emma_rt_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* cgs constants (CODATA 2018) */
static const double K_B = 1.380649e-16;              /* erg/K */
static const double E_HI = 13.6 * 1.602176634e-12;   /* "E_13.6" */

/* ------------------------------------------------------------------------------------------------
 * Closure (Eq. 22-23)
 * ---------------------------------------------------------------------------------------------- */

/* A2: chi is only described by its limits 1/3 and 1; the formula is Levermore's,
 * from the literature the paper cites.  Interior values are pinned by tests/test_oracle_literature.py:
 * chi is the Eddington factor of an isotropic field boosted by beta, f = 4 beta/(3 + beta^2), chi = (1 + 3 beta^2)/(3 + beta^2). */
double orc_chi(double f)
{
  return (3.0 + 4.0 * f * f) / (5.0 + 2.0 * sqrt(4.0 - 3.0 * f * f));
}

/* P = D N (Eq. 22);  A1: D = (1-chi)/2 I + (3chi-1)/2 n(x)n  (Eq. 23 with its two coefficients
 * un-swapped so that tr D = 1);  f = |F|/(c N) clipped to [0,1], N <= 0 -> f = 0;  |F| = 0 -> n(x)n = 0.
 * A3: c is the reduced speed of light. */
void orc_closure(const double U[4], double c, double P[9])
{
  double N = U[0];
  double Fn = sqrt(U[1] * U[1] + U[2] * U[2] + U[3] * U[3]);
  double f = 0.0;
  if (N > 0.0) {
    f = Fn / (c * N);
    if (f > 1.0) f = 1.0;
  }
  double chi = orc_chi(f);
  double nv[3] = {0.0, 0.0, 0.0};
  if (Fn > 0.0) {
    nv[0] = U[1] / Fn; nv[1] = U[2] / Fn; nv[2] = U[3] / Fn;
  }
  for (int a = 0; a < 3; a++)
    for (int b = 0; b < 3; b++) {
      double D = 0.5 * (3.0 * chi - 1.0) * nv[a] * nv[b];
      if (a == b) D += 0.5 * (1.0 - chi);
      P[3 * a + b] = D * N;
    }
}

/* ------------------------------------------------------------------------------------------------
 * Transport (Eq. 30 and 32)
 * ---------------------------------------------------------------------------------------------- */

/* flux vector in direction d:  F~_d = (F_d, c^2 P_{d,.}) */
static void flux_vector(const double U[4], double c, int d, double Ft[4])
{
  double P[9];
  orc_closure(U, c, P);
  Ft[0] = U[1 + d];
  Ft[1] = c * c * P[3 * d + 0];
  Ft[2] = c * c * P[3 * d + 1];
  Ft[3] = c * c * P[3 * d + 2];
}

/* Eq. 32:  F_{i+1/2} = (F~_i + F~_{i+1})/2 - c (U_{i+1} - U_i)/2   (L = cell i, R = cell i+1) */
static void glf_flux(const double UL[4], const double UR[4], double c, int d, double Fh[4])
{
  double FL[4], FR[4];
  flux_vector(UL, c, d, FL);
  flux_vector(UR, c, d, FR);
  for (int q = 0; q < 4; q++) Fh[q] = 0.5 * (FL[q] + FR[q]) - 0.5 * c * (UR[q] - UL[q]);
}

/* A19 -- HLL interface flux ("an implementation of the less diffusive HLL flux is also on the way";
 * nothing else is printed).  Reading: the standard HLL formula on the same flux vectors F~ as Eq. 32,
 *     F_{i+1/2} = [ l+ F~_L - l- F~_R + l+ l- (U_R - U_L) ] / (l+ - l-),
 *     l+ = max(0, lmax(U_L), lmax(U_R)),   l- = min(0, lmin(U_L), lmin(U_R)),
 * with lmin/lmax the extreme eigenvalues of dF~_d/dU for the M1 closure of Eq. 22-23 (A1, A2):
 *     l(f, mu) = c [ mu f -/+ sqrt( (2/3)(xi^2 - xi) + 2 mu^2 (2 - f^2 - xi) ) ] / xi,   xi = sqrt(4 - 3 f^2),
 * f as in the closure (clipped to [0,1], N <= 0 -> f = 0), mu = F_d/|F| (0 if |F| = 0).  l+ = -l- = c gives back Eq. 32.
 * With this flux the updated state is kept realizable: if |F'| > c N' after Eq. 30 then F' := c max(N',0) F'/|F'| (N' is not
 * touched, so photons are conserved).  Without it a beam (f = 1) is unstable: for f > 1 the clipped closure P = N n(x)n has
 * the speeds -/+c, not the (c, c) these eigenvalues give, and the upwinded flux amplifies an f > 1 perturbation by 1 + nu
 * per step (seen in the static clump test, tests/test_inflow_shadow.py).  If l+ - l- = 0 (both cells free-streaming exactly along the face) the flux is (F~_L + F~_R)/2 (= 0 there).
 * Pinned in tests against the eigenvalues of the finite-difference Jacobian of orc_closure. */
void orc_m1_wavespeeds(const double U[4], double c, int d, double* lmin, double* lmax)
{
  double N = U[0];
  double Fn = sqrt(U[1] * U[1] + U[2] * U[2] + U[3] * U[3]);
  double f = 0.0;
  if (N > 0.0) {
    f = Fn / (c * N);
    if (f > 1.0) f = 1.0;
  }
  double mu = (Fn > 0.0) ? U[1 + d] / Fn : 0.0;
  double xi = sqrt(4.0 - 3.0 * f * f);
  double rad = (2.0 / 3.0) * (xi * xi - xi) + 2.0 * mu * mu * (2.0 - f * f - xi);
  if (rad < 0.0) rad = 0.0;
  double r = sqrt(rad);
  *lmin = c * (mu * f - r) / xi;
  *lmax = c * (mu * f + r) / xi;
}

static void hll_flux(const double UL[4], const double UR[4], double c, int d, double Fh[4])
{
  double FL[4], FR[4], aL, bL, aR, bR;
  flux_vector(UL, c, d, FL);
  flux_vector(UR, c, d, FR);
  orc_m1_wavespeeds(UL, c, d, &aL, &bL);
  orc_m1_wavespeeds(UR, c, d, &aR, &bR);
  double lp = fmax(0.0, fmax(bL, bR)), lm = fmin(0.0, fmin(aL, aR));
  if (lp - lm <= 0.0) {
    for (int q = 0; q < 4; q++) Fh[q] = 0.5 * (FL[q] + FR[q]);
    return;
  }
  for (int q = 0; q < 4; q++) Fh[q] = (lp * FL[q] - lm * FR[q] + lp * lm * (UR[q] - UL[q])) / (lp - lm);
}

static void face_flux(int flux, const double UL[4], const double UR[4], double c, int d, double Fh[4])
{
  if (flux == ORC_FLUX_HLL) hll_flux(UL, UR, c, d, Fh); else glf_flux(UL, UR, c, d, Fh);
}

/* Eq. 30 summed over the three directions (A4: unsplit).  faceN[2d], faceN[2d+1] receive the N-component
 * of the flux through the -d and +d faces (used for the boundary-outflow diagnostic, A15). */
static void transport_core(int flux, double c, double dt, double dx, const double U0[4], const double Um[3][4],
                           const double Up[3][4], double out[4], double faceN[6])
{
  for (int q = 0; q < 4; q++) out[q] = U0[q];
  for (int d = 0; d < 3; d++) {
    double Fm[4], Fp[4];
    face_flux(flux, Um[d], U0, c, d, Fm);     /* F_{i-1/2} */
    face_flux(flux, U0, Up[d], c, d, Fp);     /* F_{i+1/2} */
    for (int q = 0; q < 4; q++) out[q] += (dt / dx) * (Fm[q] - Fp[q]);
    if (faceN) { faceN[2 * d] = Fm[0]; faceN[2 * d + 1] = Fp[0]; }
  }
  if (flux == ORC_FLUX_HLL) {                /* A19: keep the state realizable, |F| <= c N */
    double Fn = sqrt(out[1] * out[1] + out[2] * out[2] + out[3] * out[3]);
    double lim = c * (out[0] > 0.0 ? out[0] : 0.0);
    if (Fn > lim) for (int q = 1; q < 4; q++) out[q] *= lim / Fn;
  }
}

void orc_transport_stencil(double c, double dt, double dx, const double U0[4], const double Um[3][4],
                           const double Up[3][4], double out[4])
{
  transport_core(ORC_FLUX_GLF, c, dt, dx, U0, Um, Up, out, 0);
}

void orc_transport_stencil_flux(int flux, double c, double dt, double dx, const double U0[4], const double Um[3][4],
                                const double Up[3][4], double out[4])
{
  transport_core(flux, c, dt, dx, U0, Um, Up, out, 0);
}

/* ------------------------------------------------------------------------------------------------
 * Atomic rates (A11).  PAPER.md:312 cites Theuns et al. 1998 and Hui & Gnedin 1997 without printing
 * anything; these are literature fits restated as THE definition used by both sides.
 * Pinned by tests/test_oracle_literature.py against other sources: Osterbrock & Ferland's tabulated alpha_A, alpha_B and
 * recombination-cooling coefficients at 5e3 / 1e4 / 2e4 K, Voronov's (1997) and Cen's (1992) / Theuns et al.'s (1998)
 * collisional ionisation rate over 5e3 .. 1e6 K, Lambda_ci = 13.6 eV x beta, Cen's excitation cooling, the Rybicki &
 * Lightman free-free emissivity; a mutation test shows that a slipped exponent or prefactor in any line below fails one.
 * ---------------------------------------------------------------------------------------------- */
void orc_rates(double T, double* alphaA, double* alphaB, double* beta, double* cool_HI,
               double* cool_HII_A, double* cool_HII_B)
{
  double lam = 2.0 * 157807.0 / T;
  double aA = 1.269e-13 * pow(lam, 1.503) / pow(1.0 + pow(lam / 0.522, 0.470), 1.923);
  double aB = 2.753e-14 * pow(lam, 1.500) / pow(1.0 + pow(lam / 2.740, 0.407), 2.242);
  double be = 21.11 * pow(T, -1.5) * exp(-0.5 * lam) * pow(lam, -1.089) / pow(1.0 + pow(lam / 0.354, 0.874), 1.101);
  /* cooling, erg cm^3 s^-1 */
  double exc = 7.5e-19 * exp(-118348.0 / T) / (1.0 + sqrt(T / 1.0e5));       /* collisional excitation  */
  double cio = 2.179e-11 * be;                                               /* collisional ionisation  */
  double recA = 1.778e-29 * T * pow(lam, 1.965) / pow(1.0 + pow(lam / 0.541, 0.502), 2.697);
  double recB = 3.435e-30 * T * pow(lam, 1.970) / pow(1.0 + pow(lam / 2.250, 0.376), 3.720);
  double l10 = log10(T);
  double gff = 1.1 + 0.34 * exp(-(5.5 - l10) * (5.5 - l10) / 3.0);
  double ff = 1.42e-27 * gff * sqrt(T);                                      /* bremsstrahlung          */
  *alphaA = aA; *alphaB = aB; *beta = be;
  *cool_HI = exc + cio;
  *cool_HII_A = recA + ff;
  *cool_HII_B = recB + ff;
}

/* A10: hydrogen only, gamma = 5/3:  e = (3/2)(1+x) n0 k_B T */
double orc_temperature(double e, double x, double n0) { return e / (1.5 * (1.0 + x) * n0 * K_B); }
double orc_energy(double T, double x, double n0) { return 1.5 * (1.0 + x) * n0 * K_B * T; }

/* Lambda(n0, x, T) with the T-dependent coefficients already evaluated (n_e = x n0, n_HI = (1-x) n0, n_HII = x n0) */
static double cooling(double n0, double x, double cool_HI, double cool_HII)
{
  double ne = x * n0, nHI = (1.0 - x) * n0, nHII = x * n0;
  return ne * nHI * cool_HI + ne * nHII * cool_HII;
}

/* ------------------------------------------------------------------------------------------------
 * Thermo-chemistry, sub-cycled (Eq. 43-48; readings A5-A9)
 * ---------------------------------------------------------------------------------------------- */
int orc_chem_cell(const orc_phys* ph, double dt, double n0, double* x_io, double* e_io, double* U,
                  const double* S, orc_chem_out* out)
{
  const int G = ph->G;
  const double c = ph->c;
  double x = *x_io, e = *e_io;
  double SigE[ORC_MAX_GROUPS];
  for (int i = 0; i < G; i++) SigE[i] = ph->sigE[i] * ph->Emean[i] - ph->sigN[i] * E_HI;
  orc_chem_out o;
  memset(&o, 0, sizeof o);
  o.dtau_min = INFINITY;
  int rc = ORC_OK;

  double rem = dt;
  while (rem > 0.0) {
    /* state p */
    double T = orc_temperature(e, x, n0);
    double aA, aB, be, cHI, cHIIA, cHIIB;
    orc_rates(T, &aA, &aB, &be, &cHI, &cHIIA, &cHIIB);
    double alpha = ph->otsa ? aB : aA;            /* alpha_A := alpha_B under OTSA */
    double cHII = ph->otsa ? cHIIB : cHIIA;
    double rec_src = ph->otsa ? 0.0 : (aA - aB) * x * x * n0 * n0;       /* A6: group 1 only */

    /* first guess of the chemical step: dtau = e^p / (H^p - Lambda^p)   (A9: abs) */
    double dtau = rem;
    if (ph->thermal) {
      double H = 0.0;
      for (int i = 0; i < G; i++) H += SigE[i] * U[4 * i];
      H *= c * (1.0 - x) * n0;
      double Lam = cooling(n0, x, cHI, cHII);
      double guess = (H == Lam) ? rem : fabs(e / (H - Lam));
      if (guess < o.dtau_min) o.dtau_min = guess;
      if (guess < dtau) dtau = guess;
    }

    double N1[ORC_MAX_GROUPS], F1[ORC_MAX_GROUPS][3], x1, e1;
    int halv = 0;
    for (;;) {
      /* Eq. 43 (A5: the printed denominator lacks dtau), Eq. 44 */
      double ion = 0.0;
      for (int i = 0; i < G; i++) {
        double den = 1.0 + c * ph->sigN[i] * (1.0 - x) * n0 * dtau;
        double src = (S ? S[i] : 0.0) + (i == 0 ? rec_src : 0.0);
        N1[i] = (U[4 * i] + src * dtau) / den;
        for (int k = 0; k < 3; k++) F1[i][k] = U[4 * i + 1 + k] / den;
        ion += ph->sigN[i] * N1[i];
      }
      /* Eq. 45 as printed, multi-group via Eq. 41 (A7) */
      x1 = 1.0 - (alpha * x * x * n0 * dtau + 1.0 - x) / (1.0 + dtau * (be * x * n0 + c * ion));
      if (x1 < 0.0) x1 = 0.0;                     /* guards only; never fire in the tests */
      if (x1 > 1.0) x1 = 1.0;
      if (!ph->thermal) {
        e1 = e * (1.0 + x1) / (1.0 + x);          /* isothermal test mode: T held (A9) */
        break;
      }
      /* Eq. 46-48 (A8) */
      double heat = 0.0;
      for (int i = 0; i < G; i++) heat += SigE[i] * N1[i];
      e1 = e + dtau * (c * (1.0 - x1) * n0 * heat - cooling(n0, x1, cHI, cHII));
      /* 10 % rule */
      if (fabs(e1 - e) > ph->e_tol * e || !(e1 > 0.0)) {
        if (halv >= ph->max_halvings) { rc = ORC_ESUBCYCLE; break; }
        dtau *= 0.5;
        halv++;
        continue;
      }
      break;
    }
    o.nhalv += halv;
    if (rc != ORC_OK) break;

    /* photon bookkeeping of the accepted sub-step (A15) */
    for (int i = 0; i < G; i++) {
      o.absorbed += c * ph->sigN[i] * (1.0 - x) * n0 * dtau * N1[i];
      o.injected += (S ? S[i] : 0.0) * dtau;
    }
    o.recomb += rec_src * dtau;

    /* accept: p <- p+1 */
    for (int i = 0; i < G; i++) {
      U[4 * i] = N1[i];
      for (int k = 0; k < 3; k++) U[4 * i + 1 + k] = F1[i][k];
    }
    x = x1; e = e1;
    o.nsub++;
    if (dtau >= rem) rem = 0.0; else rem -= dtau;
    if (o.nsub >= ORC_MAX_SUBSTEPS && rem > 0.0) { rc = ORC_ESUBCYCLE; break; }
  }
  *x_io = x; *e_io = e;
  if (out) *out = o;
  return rc;
}

/* ------------------------------------------------------------------------------------------------
 * Stateful driver: coarse block + static refined levels (CRTA; A12-A15)
 * ---------------------------------------------------------------------------------------------- */
struct orc {
  int n, chemistry;
  int flux;                        /* ORC_FLUX_GLF (Eq. 32) or ORC_FLUX_HLL (A19) */
  double inflow[6][ORC_MAX_GROUPS][4]; /* A20: ghost state (N, Fx, Fy, Fz) of an ORC_BC_INFLOW face, per group */
  int bc[6];
  orc_phys ph;
  double L, dx;
  int n_levels;                    /* refined levels above the base */
  int64_t ncell[8];                /* cells per level (level 0: n^3; level l: 8*n_octs[l-1]) */
  int64_t* parent[8];              /* parent[l][oct] -> cell id on level l-1 (l >= 1) */
  int64_t* child[8];               /* child[l][cell] -> oct on level l+1, or -1 */
  double* U[2];                    /* coarse, [G][ncell0][4], double-buffered */
  int cur;
  double *n0[8], *x[8], *e[8];
  uint32_t* subc[8];               /* accepted | halvings<<16 of the last step */
  double* S[8];                    /* per level, [ncell][G] source density, or NULL */
  int64_t n_src;
  int64_t* src_cell; int* src_level;
  double t_sim;
  int64_t cnt_transport_cells[8];  /* cells swept by the transport engine, per level (CRTA: level 0 only) */
  int64_t cnt_chem_cells[8];       /* leaf cells swept by the chemistry engine, per level */
  /* standard (non-CRTA) AMR transport, reading A21; see the section at the end of this file */
  int amr;                         /* 0: CRTA (default); 1: level-by-level transport on every level */
  double* Ul[8];                   /* l >= 1: radiation of level l, [G][ncell_l][4] (level 0 lives in U[cur]) */
  double* dep[8];                  /* per level: change deposited into leaf cells by the fluxes of the finer level */
  int32_t* coord[8];               /* [ncell_l][3] integer cell coordinates on level l, in [0, n 2^l) */
};

int orc_set_flux(orc* o, int flux)
{
  if (!o || (flux != ORC_FLUX_GLF && flux != ORC_FLUX_HLL)) return ORC_EINVAL;
  o->flux = flux;
  return ORC_OK;
}

/* A20: prescribed ghost state of an inflow face (face = -x,+x,-y,+y,-z,+z), cgs */
int orc_set_inflow(orc* o, int face, int group, const double U[4])
{
  if (!o || face < 0 || face > 5 || group < 0 || group >= o->ph.G || !U) return ORC_EINVAL;
  if (o->bc[face] != ORC_BC_INFLOW) return ORC_EINVAL;
  for (int q = 0; q < 4; q++) o->inflow[face][group][q] = U[q];
  return ORC_OK;
}

int orc_threads(void)
{
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

int64_t orc_level_cells(const orc* o, int level) { return (level < 0 || level > o->n_levels) ? -1 : o->ncell[level]; }

void orc_free(orc* o)
{
  if (!o) return;
  free(o->U[0]); free(o->U[1]);
  for (int l = 0; l < 8; l++) {
    free(o->parent[l]); free(o->child[l]); free(o->n0[l]); free(o->x[l]); free(o->e[l]);
    free(o->subc[l]); free(o->S[l]);
  }
  free(o->src_cell); free(o->src_level);
  for (int l = 0; l < 8; l++) { free(o->Ul[l]); free(o->dep[l]); free(o->coord[l]); }
  free(o);
}

/* arithmetic mean of the 8 children of an oct (A14), summed pairwise along x, then y, then z
 * (child index = ix + 2 iy + 4 iz), so that 8 identical children average to exactly their common value */
static double mean8(const double v[8])
{
  return (((v[0] + v[1]) + (v[2] + v[3])) + ((v[4] + v[5]) + (v[6] + v[7]))) / 8.0;
}

/* bottom-up: split cell := mean of its 8 children */
static void restrict_scalar(orc* o, double** a)
{
  for (int l = o->n_levels; l >= 1; l--) {
    int64_t noct = o->ncell[l] / 8;
    for (int64_t oc = 0; oc < noct; oc++) a[l - 1][o->parent[l][oc]] = mean8(a[l] + 8 * oc);
  }
}

orc* orc_create(int n, const int bc[6], int chemistry, const orc_phys* ph, double box_len,
                int n_levels, const int64_t* n_octs, const int64_t* const* parent,
                const float* const* U0, const float* const* n0, const float* const* x, const float* const* T)
{
  if (n < 1 || !ph || ph->G < 1 || ph->G > ORC_MAX_GROUPS || n_levels < 0 || n_levels > 7) return 0;
  orc* o = (orc*)calloc(1, sizeof(orc));
  if (!o) return 0;
  o->n = n; o->chemistry = chemistry; o->ph = *ph; o->L = box_len; o->dx = box_len / n;
  memcpy(o->bc, bc, sizeof o->bc);
  o->n_levels = n_levels;
  o->ncell[0] = (int64_t)n * n * n;
  for (int l = 1; l <= n_levels; l++) o->ncell[l] = 8 * n_octs[l - 1];
  const int G = ph->G;
  for (int b = 0; b < 2; b++) {
    o->U[b] = (double*)calloc((size_t)G * o->ncell[0] * 4, sizeof(double));
    if (!o->U[b]) { orc_free(o); return 0; }
  }
  for (int l = 0; l <= n_levels; l++) {
    int64_t nc = o->ncell[l];
    size_t na = nc > 0 ? (size_t)nc : 1;
    o->n0[l] = (double*)calloc(na, sizeof(double));
    o->x[l] = (double*)calloc(na, sizeof(double));
    o->e[l] = (double*)calloc(na, sizeof(double));
    o->subc[l] = (uint32_t*)calloc(na, sizeof(uint32_t));
    o->child[l] = (int64_t*)malloc(na * sizeof(int64_t));
    if (!o->n0[l] || !o->x[l] || !o->e[l] || !o->subc[l] || !o->child[l]) { orc_free(o); return 0; }
    for (int64_t i = 0; i < nc; i++) o->child[l][i] = -1;
  }
  for (int l = 1; l <= n_levels; l++) {
    int64_t noct = n_octs[l - 1];
    o->parent[l] = (int64_t*)malloc((noct > 0 ? noct : 1) * sizeof(int64_t));
    if (!o->parent[l]) { orc_free(o); return 0; }
    for (int64_t oc = 0; oc < noct; oc++) {
      int64_t p = parent[l - 1][oc];
      if (p < 0 || p >= o->ncell[l - 1] || o->child[l - 1][p] != -1) { orc_free(o); return 0; }
      o->parent[l][oc] = p;
      o->child[l - 1][p] = oc;
    }
  }
  /* inputs are fp32 (the same bytes the library gets); held in fp64 from here on */
  if (U0)
    for (int g = 0; g < G; g++)
      if (U0[g])
        for (int64_t i = 0; i < o->ncell[0] * 4; i++) o->U[0][(size_t)g * o->ncell[0] * 4 + i] = (double)U0[g][i];
  for (int l = 0; l <= n_levels; l++)
    for (int64_t i = 0; i < o->ncell[l]; i++) {
      o->n0[l][i] = (double)n0[l][i];
      o->x[l][i] = (double)x[l][i];
      o->e[l][i] = orc_energy((double)T[l][i], (double)x[l][i], (double)n0[l][i]);   /* A10 */
    }
  /* split cells hold the children mean (input entries of split cells are ignored) */
  restrict_scalar(o, o->n0);
  restrict_scalar(o, o->x);
  restrict_scalar(o, o->e);
  return o;
}

/* A12: NGP into the leaf cell containing the position; S_g = Q_g / dV_leaf; same-cell sources add */
int orc_set_sources(orc* o, int64_t n_src, const double* pos, const double* Q)
{
  const int G = o->ph.G;
  if (n_src < 0) return ORC_EINVAL;
  for (int64_t s = 0; s < n_src; s++) {
    for (int k = 0; k < 3; k++)
      if (!(pos[3 * s + k] >= 0.0 && pos[3 * s + k] < 1.0)) return ORC_EINVAL;
    for (int g = 0; g < G; g++)
      if (!(Q[s * G + g] >= 0.0) || isinf(Q[s * G + g])) return ORC_EINVAL;
  }
  for (int l = 0; l <= o->n_levels; l++) { free(o->S[l]); o->S[l] = 0; }
  free(o->src_cell); free(o->src_level);
  o->src_cell = (int64_t*)malloc((n_src > 0 ? n_src : 1) * sizeof(int64_t));
  o->src_level = (int*)malloc((n_src > 0 ? n_src : 1) * sizeof(int));
  o->n_src = n_src;
  for (int64_t s = 0; s < n_src; s++) {
    const double* p = pos + 3 * s;
    int n = o->n;
    double fx = p[0] * n, fy = p[1] * n, fz = p[2] * n;
    int ix = (int)floor(fx), iy = (int)floor(fy), iz = (int)floor(fz);
    if (ix >= n) ix = n - 1;
    if (iy >= n) iy = n - 1;
    if (iz >= n) iz = n - 1;
    int lvl = 0;
    int64_t cell = ix + (int64_t)n * (iy + (int64_t)n * iz);
    double ox = fx - ix, oy = fy - iy, oz = fz - iz;          /* offset inside the cell, [0,1) */
    while (lvl < o->n_levels && o->child[lvl][cell] >= 0) {
      int64_t oc = o->child[lvl][cell];
      int cx = ox >= 0.5, cy = oy >= 0.5, cz = oz >= 0.5;
      ox = 2.0 * ox - cx; oy = 2.0 * oy - cy; oz = 2.0 * oz - cz;
      cell = 8 * oc + (cx + 2 * cy + 4 * cz);
      lvl++;
    }
    if (!o->S[lvl]) o->S[lvl] = (double*)calloc((size_t)o->ncell[lvl] * G, sizeof(double));
    double dxl = o->dx / (double)(1 << lvl);
    double dV = dxl * dxl * dxl;
    for (int g = 0; g < G; g++) o->S[lvl][cell * G + g] += Q[s * G + g] / dV;
    o->src_cell[s] = cell; o->src_level[s] = lvl;
  }
  return ORC_OK;
}

int64_t orc_source_cell(const orc* o, int64_t i, int* level)
{
  if (i < 0 || i >= o->n_src) return -1;
  if (level) *level = o->src_level[i];
  return o->src_cell[i];
}

/* ghost value of the neighbour of (i,j,k) in direction d, side s (A13) */
static void neighbour(const orc* o, const double* Ug, int g, int i, int j, int k, int d, int s, double out[4])
{
  const int n = o->n;
  int idx[3] = {i, j, k};
  idx[d] += s;
  int flip = 0;
  if (idx[d] < 0 || idx[d] >= n) {
    int bc = o->bc[2 * d + (s > 0 ? 1 : 0)];
    if (bc == ORC_BC_PERIODIC) idx[d] = (idx[d] + n) % n;
    else if (bc == ORC_BC_INFLOW) {          /* A20: the ghost holds the prescribed incoming state */
      const double* q = o->inflow[2 * d + (s > 0 ? 1 : 0)][g];
      for (int c = 0; c < 4; c++) out[c] = q[c];
      return;
    }
    else {                                   /* transmissive: copy self; reflective: + flux inversion */
      idx[d] = (d == 0 ? i : d == 1 ? j : k);
      flip = (bc == ORC_BC_REFLECTIVE);
    }
  }
  const double* p = Ug + 4 * ((size_t)idx[0] + (size_t)n * (idx[1] + (size_t)n * idx[2]));
  for (int q = 0; q < 4; q++) out[q] = p[q];
  if (flip) out[1 + d] = -out[1 + d];       /* face-normal component only (A13) */
}

typedef struct { double absorbed, injected, recomb, total, dtau_min; int64_t nsub, nsub_max, nhalv, leaves[8]; int rc; } acc_t;

static void acc_init(acc_t* a) { memset(a, 0, sizeof *a); a->dtau_min = INFINITY; }
static void acc_add(acc_t* a, const acc_t* b)
{
  a->absorbed += b->absorbed; a->injected += b->injected; a->recomb += b->recomb; a->total += b->total;
  if (b->dtau_min < a->dtau_min) a->dtau_min = b->dtau_min;
  a->nsub += b->nsub; a->nhalv += b->nhalv;
  for (int l = 0; l < 8; l++) a->leaves[l] += b->leaves[l];
  if (b->nsub_max > a->nsub_max) a->nsub_max = b->nsub_max;
  if (b->rc != ORC_OK && a->rc == ORC_OK) a->rc = b->rc;
}

/* chemistry of one LEAF cell of level l with incoming radiation Uin[G][4]; result in Uout */
static void leaf_update(orc* o, double dt, int l, int64_t cell, const double* Uin, double* Uout, acc_t* a)
{
  const int G = o->ph.G;
  double dxl = o->dx / (double)(1 << l), dV = dxl * dxl * dxl;
  memcpy(Uout, Uin, sizeof(double) * 4 * G);
  a->leaves[l]++;
  const double* S = o->S[l] ? o->S[l] + cell * G : 0;
  if (o->chemistry) {
    orc_chem_out co;
    int rc = orc_chem_cell(&o->ph, dt, o->n0[l][cell], &o->x[l][cell], &o->e[l][cell], Uout, S, &co);
    a->absorbed += co.absorbed * dV; a->injected += co.injected * dV; a->recomb += co.recomb * dV;
    if (co.dtau_min < a->dtau_min) a->dtau_min = co.dtau_min;
    a->nsub += co.nsub; a->nhalv += co.nhalv;
    if (co.nsub > a->nsub_max) a->nsub_max = co.nsub;
    if (rc != ORC_OK && a->rc == ORC_OK) a->rc = rc;
    unsigned ns = co.nsub > 65535 ? 65535u : (unsigned)co.nsub, nh = co.nhalv > 65535 ? 65535u : (unsigned)co.nhalv;
    o->subc[l][cell] = ns | (nh << 16);
  } else if (S) {
    /* chemistry off: Eq. 43 degenerates to N += S dt, F unchanged (A9) */
    for (int g = 0; g < G; g++) { Uout[4 * g] += S[g] * dt; a->injected += S[g] * dt * dV; }
  }
  for (int g = 0; g < G; g++) a->total += Uout[4 * g] * dV;
}

/* CRTA (A14): a split cell injects the incoming (coarse) radiation unchanged into its 8
 * children, each child is updated (recursively), and the split cell takes the mean of the children
 * for N_g, F_g, x, e. */
static void cell_update(orc* o, double dt, int l, int64_t cell, const double* Uin, double* Uout, acc_t* a)
{
  const int G = o->ph.G;
  int64_t oc = (l < o->n_levels) ? o->child[l][cell] : -1;
  if (oc < 0) { leaf_update(o, dt, l, cell, Uin, Uout, a); return; }
  double Uc[8][4 * ORC_MAX_GROUPS], v[8];
  for (int k = 0; k < 8; k++) cell_update(o, dt, l + 1, 8 * oc + k, Uin, Uc[k], a);
  for (int q = 0; q < 4 * G; q++) {
    for (int k = 0; k < 8; k++) v[k] = Uc[k][q];
    Uout[q] = mean8(v);
  }
  o->x[l][cell] = mean8(o->x[l + 1] + 8 * oc);
  o->e[l][cell] = mean8(o->e[l + 1] + 8 * oc);
  o->subc[l][cell] = 0;
}

static int amr_step(orc* o, double dt, int n_steps, orc_diag* diag);

int orc_step(orc* o, double dt, int n_steps, orc_diag* diag)
{
  if (o->amr) return amr_step(o, dt, n_steps, diag);
  const int n = o->n, G = o->ph.G;
  const int64_t nc = o->ncell[0];
  const double c = o->ph.c, dx = o->dx;
  if (!(dt > 0.0) || n_steps < 0) return ORC_EINVAL;
  if (3.0 * c * dt > dx * (1.0 + 1e-12)) return ORC_ECFL;          /* A4: dt <= dx/(3c) */
  int rc_all = ORC_OK;
  orc_diag dg;
  memset(&dg, 0, sizeof dg);
  acc_t* slab = (acc_t*)malloc(sizeof(acc_t) * n);
  double* outflow = (double*)malloc(sizeof(double) * n);
  if (!slab || !outflow) { free(slab); free(outflow); return ORC_ENOMEM; }

  for (int step = 0; step < n_steps; step++) {
    const double* Uold = o->U[o->cur];
    double* Unew = o->U[1 - o->cur];
    /* 1-2. ghosts + transport on the coarse level, each group independently */
#pragma omp parallel for schedule(static)
    for (int k = 0; k < n; k++) {
      double of = 0.0;
      for (int g = 0; g < G; g++) {
        const double* Ug = Uold + (size_t)g * nc * 4;
        double* Vg = Unew + (size_t)g * nc * 4;
        for (int j = 0; j < n; j++)
          for (int i = 0; i < n; i++) {
            size_t id = (size_t)i + (size_t)n * (j + (size_t)n * k);
            double Um[3][4], Up[3][4], faceN[6];
            for (int d = 0; d < 3; d++) {
              neighbour(o, Ug, g, i, j, k, d, -1, Um[d]);
              neighbour(o, Ug, g, i, j, k, d, +1, Up[d]);
            }
            transport_core(o->flux, c, dt, dx, Ug + 4 * id, Um, Up, Vg + 4 * id, faceN);
            /* net photon flux through non-periodic box faces (A15) */
            int idx[3] = {i, j, k};
            for (int d = 0; d < 3; d++) {
              if (idx[d] == 0 && o->bc[2 * d] != ORC_BC_PERIODIC) of -= faceN[2 * d] * dx * dx * dt;
              if (idx[d] == n - 1 && o->bc[2 * d + 1] != ORC_BC_PERIODIC) of += faceN[2 * d + 1] * dx * dx * dt;
            }
          }
      }
      outflow[k] = of;
    }
    o->cur = 1 - o->cur;
    double* U = o->U[o->cur];

    /* 3-5. inject -> leaf chemistry -> restrict, cell by cell (in place on the new coarse buffer) */
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n; k++) {
      acc_t a;
      acc_init(&a);
      double Uin[4 * ORC_MAX_GROUPS], Uout[4 * ORC_MAX_GROUPS];
      for (int64_t id = (int64_t)k * n * n; id < (int64_t)(k + 1) * n * n; id++) {
        for (int g = 0; g < G; g++)
          for (int q = 0; q < 4; q++) Uin[4 * g + q] = U[((size_t)g * nc + id) * 4 + q];
        cell_update(o, dt, 0, id, Uin, Uout, &a);
        for (int g = 0; g < G; g++)
          for (int q = 0; q < 4; q++) U[((size_t)g * nc + id) * 4 + q] = Uout[4 * g + q];
      }
      slab[k] = a;
    }

    /* 6. diagnostics, serial in slab order */
    acc_t tot;
    acc_init(&tot);
    double of = 0.0;
    for (int k = 0; k < n; k++) { acc_add(&tot, &slab[k]); of += outflow[k]; }
    if (tot.rc != ORC_OK && rc_all == ORC_OK) rc_all = tot.rc;
    o->t_sim += dt;
    o->cnt_transport_cells[0] += nc;
    for (int l = 0; l < 8; l++) o->cnt_chem_cells[l] += tot.leaves[l];
    dg.photons_total = tot.total; dg.photons_injected = tot.injected; dg.photons_absorbed = tot.absorbed;
    dg.photons_recomb_emitted = tot.recomb; dg.photons_outflow = of; dg.dtau_min = tot.dtau_min;
    dg.subcycles_total = tot.nsub; dg.subcycles_max = tot.nsub_max; dg.halvings_total = tot.nhalv;
    dg.t_sim = o->t_sim;
  }
  free(slab); free(outflow);

  /* non-finite scan of the final state */
  int64_t bad = 0;
  for (int64_t i = 0; i < (int64_t)G * nc * 4; i++) bad += !isfinite(o->U[o->cur][i]);
  for (int l = 0; l <= o->n_levels; l++)
    for (int64_t i = 0; i < o->ncell[l]; i++) bad += !isfinite(o->x[l][i]) + !isfinite(o->e[l][i]);
  dg.n_nonfinite = bad;
  if (n_steps == 0) {
    double tot = 0.0, dV = dx * dx * dx;
    for (int64_t i = 0; i < (int64_t)G * nc; i++) tot += o->U[o->cur][4 * i] * dV;
    dg.photons_total = tot; dg.t_sim = o->t_sim; dg.dtau_min = INFINITY;
  }
  if (diag) *diag = dg;
  if (bad && rc_all == ORC_OK) rc_all = ORC_ENONFINITE;
  return rc_all;
}

void orc_counters(const orc* o, int64_t transport_cells[8], int64_t chem_cells[8])
{
  for (int l = 0; l < 8; l++) { transport_cells[l] = o->cnt_transport_cells[l]; chem_cells[l] = o->cnt_chem_cells[l]; }
}

int orc_read(const orc* o, int field, int level, int group, double* dst, int64_t n_dst)
{
  if (level < 0 || level > o->n_levels) return ORC_EINVAL;
  const int64_t nc = o->ncell[level];
  const int G = o->ph.G;
  if (field == ORC_F_U || field == ORC_F_N || field == ORC_F_F) {
    if ((level != 0 && !o->amr) || group < 0 || group >= G) return ORC_EINVAL;
    const double* Ug = (level == 0 ? o->U[o->cur] : o->Ul[level]) + (size_t)group * nc * 4;
    int per = field == ORC_F_U ? 4 : field == ORC_F_N ? 1 : 3;
    if (n_dst < nc * per) return ORC_EINVAL;
    for (int64_t i = 0; i < nc; i++) {
      if (field == ORC_F_U) for (int q = 0; q < 4; q++) dst[4 * i + q] = Ug[4 * i + q];
      else if (field == ORC_F_N) dst[i] = Ug[4 * i];
      else for (int q = 0; q < 3; q++) dst[3 * i + q] = Ug[4 * i + 1 + q];
    }
    return ORC_OK;
  }
  if (n_dst < nc) return ORC_EINVAL;
  for (int64_t i = 0; i < nc; i++) {
    switch (field) {
      case ORC_F_X: dst[i] = o->x[level][i]; break;
      case ORC_F_XNEUTRAL: dst[i] = 1.0 - o->x[level][i]; break;
      case ORC_F_E: dst[i] = o->e[level][i]; break;
      case ORC_F_N0: dst[i] = o->n0[level][i]; break;
      case ORC_F_T: dst[i] = orc_temperature(o->e[level][i], o->x[level][i], o->n0[level][i]); break;
      case ORC_F_SUBCYCLES: dst[i] = (double)o->subc[level][i]; break;
      default: return ORC_EINVAL;
    }
  }
  return ORC_OK;
}

/* ================================================================================================
 * Standard (non-CRTA) AMR transport -- SURVEY.md 8f NEXT-2, reading A21 of DESIGN.md
 * (Eq. 49-51, Fig. 2-3; resolution jumps in the gather).
 *
 * Every cell of every level carries (N_g, F_g).  Levels are advanced recursively, finest first,
 * dt_l = dt_{l-1}/2 (Eq. 50-51 with equal halves):
 *
 *     advance(l, dt):   if level l+1 has octs: advance(l+1, dt/2); advance(l+1, dt/2)
 *                       transport of the LEAF cells of level l over dt     (Eq. 30, 32 / A19)
 *                       chemistry of the LEAF cells of level l over dt     (Eq. 43-48)
 *                       split cells of level l := mean of their 8 children (N, F, x, e, A14)
 *
 * Faces of a leaf cell of level l (the sequence (i)-(iii) of Fig. 3):
 *   - neighbour is a leaf of level l: the flux of Eq. 32 between the two states at the start of the step;
 *   - neighbour of level l is SPLIT: nothing is computed here; the cell has already been "temporarily updated"
 *     by the fluxes of the two sub-steps of the 4 fine cells behind that face (kept in dep[l] until now);
 *   - neighbour does not exist on level l (a leaf of level l-1; jumps are <= 1): the missing cell
 *     is "interpolated linearly from coarse data at the position of the fine virtual cell":
 *         U_ghost = U_c + sum_a (+-1/4) Delta_a,   Delta_a = minmod(U_c - U_{c-a}, U_{c+a} - U_c)
 *     per component, with U_c the coarse leaf AT THE START OF ITS OWN STEP (Fig. 3: F(U^{p+1/2}_{l+1}, U^p_l)),
 *     c+-a its neighbours on level l-1 (a split one holds its children mean, one that is coarser still is
 *     taken piecewise constant, one outside the box follows the boundary rule of A13/A20 applied to c), the sign
 *     given by which half of c the virtual cell sits in.  MinMod is the limiter the paper names for its slopes
 *     (PAPER.md:167); it keeps the ghost inside the range of the coarse values, so N_ghost >= 0.
 *     The same flux, times dt_l dx_l^2 / dx_{l-1}^3, is deposited into c with the opposite sign.
 * Box faces follow A13 / A20 on every level.  The CFL number c dt_l / dx_l is the same on every level.
 * ============================================================================================== */

static double* amr_U(orc* o, int l) { return l == 0 ? o->U[o->cur] : o->Ul[l]; }

static double minmod(double a, double b)
{
  if (a * b <= 0.0) return 0.0;
  return (fabs(a) < fabs(b)) ? a : b;
}

/* the cell of level <= l that covers the level-l coordinates (ci, cj, ck); *lf = its level */
static int64_t amr_find(const orc* o, int l, int ci, int cj, int ck, int* lf)
{
  const int n = o->n;
  int64_t cell = (ci >> l) + (int64_t)n * ((cj >> l) + (int64_t)n * (ck >> l));
  int m = 0;
  while (m < l) {
    int64_t oc = o->child[m][cell];
    if (oc < 0) break;
    m++;
    int sh = l - m;
    cell = 8 * oc + (((ci >> sh) & 1) + 2 * ((cj >> sh) & 1) + 4 * ((ck >> sh) & 1));
  }
  *lf = m;
  return cell;
}

/* state of group g seen across face (d, s) of the level-l cell with coordinates co[]: kind = 0 a cell of level l
 * (or a box-face ghost), 1 a split cell of level l (no flux here), 2 a coarser leaf (out = piecewise-constant
 * value; the caller interpolates).  *nb = the neighbour cell, *lnb its level (box-face ghosts: -1). */
static int amr_neighbour(orc* o, int l, int g, const int32_t co[3], int64_t self, int d, int s, double out[4],
                         int64_t* nb, int* lnb)
{
  const int nl = o->n << l;
  int c[3] = {co[0], co[1], co[2]};
  c[d] += s;
  *nb = -1; *lnb = -1;
  if (c[d] < 0 || c[d] >= nl) {
    int bc = o->bc[2 * d + (s > 0 ? 1 : 0)];
    if (bc == ORC_BC_PERIODIC) c[d] = (c[d] + nl) % nl;
    else if (bc == ORC_BC_INFLOW) {
      for (int q = 0; q < 4; q++) out[q] = o->inflow[2 * d + (s > 0 ? 1 : 0)][g][q];
      return 0;
    } else {
      const double* p = amr_U(o, l) + ((size_t)g * o->ncell[l] + self) * 4;
      for (int q = 0; q < 4; q++) out[q] = p[q];
      if (bc == ORC_BC_REFLECTIVE) out[1 + d] = -out[1 + d];
      return 0;
    }
  }
  int lf;
  int64_t cell = amr_find(o, l, c[0], c[1], c[2], &lf);
  const double* p = amr_U(o, lf) + ((size_t)g * o->ncell[lf] + cell) * 4;
  for (int q = 0; q < 4; q++) out[q] = p[q];
  *nb = cell; *lnb = lf;
  if (lf < l) return 2;
  return (l < o->n_levels && o->child[l][cell] >= 0) ? 1 : 0;
}

/* the virtual level-l cell at coordinates v[] inside the level-(l-1) leaf c, linearly interpolated */
static void amr_ghost(orc* o, int l, int g, const int v[3], int64_t c, double out[4])
{
  const int lc = l - 1;
  const double* Uc = amr_U(o, lc) + ((size_t)g * o->ncell[lc] + c) * 4;
  const int32_t* cc = o->coord[lc] + 3 * c;
  for (int q = 0; q < 4; q++) out[q] = Uc[q];
  for (int a = 0; a < 3; a++) {
    double Um[4], Up[4];
    int64_t nb; int lnb;
    amr_neighbour(o, lc, g, cc, c, a, -1, Um, &nb, &lnb);
    amr_neighbour(o, lc, g, cc, c, a, +1, Up, &nb, &lnb);
    double sgn = (v[a] & 1) ? 0.25 : -0.25;
    for (int q = 0; q < 4; q++) out[q] += sgn * minmod(Uc[q] - Um[q], Up[q] - Uc[q]);
  }
}

/* transport of the leaf cells of level l over dt (Eq. 30); returns the net outflow through non-periodic box faces */
static double amr_transport_level(orc* o, int l, double dt)
{
  const int G = o->ph.G;
  const int64_t nc = o->ncell[l];
  const double c = o->ph.c, dxl = o->dx / (double)(1 << l);
  const int nl = o->n << l;
  double* U = amr_U(o, l);
  double* Un = (double*)malloc(sizeof(double) * (size_t)G * nc * 4);
  memcpy(Un, U, sizeof(double) * (size_t)G * nc * 4);
  double of = 0.0;
  for (int g = 0; g < G; g++)
    for (int64_t cell = 0; cell < nc; cell++) {
      if (l < o->n_levels && o->child[l][cell] >= 0) continue;            /* split: restricted later */
      const int32_t* co = o->coord[l] + 3 * cell;
      const double* U0 = U + ((size_t)g * nc + cell) * 4;
      double out[4];
      for (int q = 0; q < 4; q++) out[q] = U0[q];
      for (int d = 0; d < 3; d++) {
        double Fh[2][4];                                                  /* F_{i-1/2}, F_{i+1/2} */
        for (int side = 0; side < 2; side++) {
          const int s = side ? +1 : -1;
          double Unb[4];
          int64_t nb; int lnb;
          int kind = amr_neighbour(o, l, g, co, cell, d, s, Unb, &nb, &lnb);
          if (kind == 1) { for (int q = 0; q < 4; q++) Fh[side][q] = 0.0; continue; }   /* (iii): fine fluxes only */
          if (kind == 2) {
            int v[3] = {co[0], co[1], co[2]};
            v[d] = (v[d] + s + nl) % nl;
            amr_ghost(o, l, g, v, nb, Unb);
          }
          if (side == 0) face_flux(o->flux, Unb, U0, c, d, Fh[0]); else face_flux(o->flux, U0, Unb, c, d, Fh[1]);
          if (kind == 2) {                                                /* (i)-(ii): the same flux updates the coarse cell */
            double* dp = o->dep[l - 1] + ((size_t)g * o->ncell[l - 1] + nb) * 4;
            double w = dt / (8.0 * dxl);                                  /* dt dx_l^2 / (2 dx_l)^3 */
            for (int q = 0; q < 4; q++) dp[q] += (side ? +w : -w) * Fh[side][q];
          }
          if (lnb < 0 && o->bc[2 * d + side] != ORC_BC_PERIODIC)          /* box face (A15) */
            of += (side ? +1.0 : -1.0) * Fh[side][0] * dxl * dxl * dt;
        }
        for (int q = 0; q < 4; q++) out[q] += (dt / dxl) * (Fh[0][q] - Fh[1][q]);
      }
      double* dp = o->dep[l] + ((size_t)g * nc + cell) * 4;
      for (int q = 0; q < 4; q++) { out[q] += dp[q]; dp[q] = 0.0; }
      if (o->flux == ORC_FLUX_HLL) {                                      /* A19: keep the state realizable */
        double Fn = sqrt(out[1] * out[1] + out[2] * out[2] + out[3] * out[3]);
        double lim = c * (out[0] > 0.0 ? out[0] : 0.0);
        if (Fn > lim) for (int q = 1; q < 4; q++) out[q] *= lim / Fn;
      }
      for (int q = 0; q < 4; q++) Un[((size_t)g * nc + cell) * 4 + q] = out[q];
    }
  memcpy(U, Un, sizeof(double) * (size_t)G * nc * 4);
  free(Un);
  o->cnt_transport_cells[l] += nc;
  return of;
}

/* chemistry of the leaf cells of level l over dt (Eq. 43-48), in place */
static void amr_chem_level(orc* o, int l, double dt, acc_t* a)
{
  const int G = o->ph.G;
  const int64_t nc = o->ncell[l];
  double* U = amr_U(o, l);
  double Uin[4 * ORC_MAX_GROUPS], Uout[4 * ORC_MAX_GROUPS];
  for (int64_t cell = 0; cell < nc; cell++) {
    if (l < o->n_levels && o->child[l][cell] >= 0) { o->subc[l][cell] = 0; continue; }
    for (int g = 0; g < G; g++)
      for (int q = 0; q < 4; q++) Uin[4 * g + q] = U[((size_t)g * nc + cell) * 4 + q];
    leaf_update(o, dt, l, cell, Uin, Uout, a);
    for (int g = 0; g < G; g++)
      for (int q = 0; q < 4; q++) U[((size_t)g * nc + cell) * 4 + q] = Uout[4 * g + q];
  }
}

/* split cells of level l := mean of their 8 children (N, F, x, e) */
static void amr_restrict_level(orc* o, int l)
{
  if (l >= o->n_levels) return;
  const int G = o->ph.G;
  const int64_t noct = o->ncell[l + 1] / 8;
  double v[8];
  for (int64_t oc = 0; oc < noct; oc++) {
    int64_t p = o->parent[l + 1][oc];
    for (int g = 0; g < G; g++)
      for (int q = 0; q < 4; q++) {
        for (int k = 0; k < 8; k++) v[k] = o->Ul[l + 1][((size_t)g * o->ncell[l + 1] + 8 * oc + k) * 4 + q];
        amr_U(o, l)[((size_t)g * o->ncell[l] + p) * 4 + q] = mean8(v);
      }
    o->x[l][p] = mean8(o->x[l + 1] + 8 * oc);
    o->e[l][p] = mean8(o->e[l + 1] + 8 * oc);
  }
}

static void amr_advance(orc* o, int l, double dt, acc_t* a, double* outflow)
{
  if (l < o->n_levels && o->ncell[l + 1] > 0) {
    amr_advance(o, l + 1, 0.5 * dt, a, outflow);
    amr_advance(o, l + 1, 0.5 * dt, a, outflow);
  }
  *outflow += amr_transport_level(o, l, dt);
  amr_chem_level(o, l, dt, a);
  amr_restrict_level(o, l);
}

static int amr_step(orc* o, double dt, int n_steps, orc_diag* diag)
{
  const int G = o->ph.G;
  if (!(dt > 0.0) || n_steps < 0) return ORC_EINVAL;
  if (3.0 * o->ph.c * dt > o->dx * (1.0 + 1e-12)) return ORC_ECFL;      /* A4; the same CFL number on every level */
  int rc_all = ORC_OK;
  orc_diag dg;
  memset(&dg, 0, sizeof dg);
  dg.dtau_min = INFINITY;
  for (int step = 0; step < n_steps; step++) {
    acc_t a;
    acc_init(&a);
    double of = 0.0;
    amr_advance(o, 0, dt, &a, &of);
    if (a.rc != ORC_OK && rc_all == ORC_OK) rc_all = a.rc;
    o->t_sim += dt;
    for (int l = 0; l < 8; l++) o->cnt_chem_cells[l] += a.leaves[l];
    dg.photons_injected = a.injected; dg.photons_absorbed = a.absorbed; dg.photons_recomb_emitted = a.recomb;
    dg.photons_outflow = of; dg.dtau_min = a.dtau_min;
    dg.subcycles_total = a.nsub; dg.subcycles_max = a.nsub_max; dg.halvings_total = a.nhalv;
  }
  /* photons on the leaves, and the non-finite scan */
  double tot = 0.0;
  int64_t bad = 0;
  for (int l = 0; l <= o->n_levels; l++) {
    double dxl = o->dx / (double)(1 << l), dV = dxl * dxl * dxl;
    const double* U = amr_U(o, l);
    for (int64_t cell = 0; cell < o->ncell[l]; cell++) {
      int leaf = !(l < o->n_levels && o->child[l][cell] >= 0);
      for (int g = 0; g < G; g++) {
        const double* p = U + ((size_t)g * o->ncell[l] + cell) * 4;
        if (leaf) tot += p[0] * dV;
        for (int q = 0; q < 4; q++) bad += !isfinite(p[q]);
      }
      bad += !isfinite(o->x[l][cell]) + !isfinite(o->e[l][cell]);
    }
  }
  dg.photons_total = tot; dg.n_nonfinite = bad; dg.t_sim = o->t_sim;
  if (diag) *diag = dg;
  if (bad && rc_all == ORC_OK) rc_all = ORC_ENONFINITE;
  return rc_all;
}

/* Switch to the standard AMR transport (A21).  Computes the cell coordinates of every level, checks that
 * resolution jumps across faces are <= 1 (ORC_EINVAL otherwise) and gives every refined cell the
 * radiation of its parent ("physical quantities are straightforwardly injected from coarse values"). */
int orc_set_amr_transport(orc* o, int on)
{
  if (!o) return ORC_EINVAL;
  if (!on) { o->amr = 0; return ORC_OK; }
  const int G = o->ph.G, n = o->n;
  for (int l = 0; l <= o->n_levels; l++) {
    const int64_t nc = o->ncell[l];
    size_t na = nc > 0 ? (size_t)nc : 1;
    free(o->coord[l]); free(o->dep[l]);
    o->coord[l] = (int32_t*)malloc(na * 3 * sizeof(int32_t));
    o->dep[l] = (double*)calloc(na * 4 * G, sizeof(double));
    if (l >= 1) { free(o->Ul[l]); o->Ul[l] = (double*)calloc(na * 4 * G, sizeof(double)); }
    if (!o->coord[l] || !o->dep[l] || (l >= 1 && !o->Ul[l])) return ORC_ENOMEM;
    if (l == 0) {
      for (int64_t id = 0; id < nc; id++) {
        o->coord[0][3 * id] = (int32_t)(id % n);
        o->coord[0][3 * id + 1] = (int32_t)((id / n) % n);
        o->coord[0][3 * id + 2] = (int32_t)(id / ((int64_t)n * n));
      }
    } else {
      for (int64_t oc = 0; oc < nc / 8; oc++) {
        int64_t p = o->parent[l][oc];
        const int32_t* pc = o->coord[l - 1] + 3 * p;
        for (int k = 0; k < 8; k++) {
          int32_t* cc = o->coord[l] + 3 * (8 * oc + k);
          cc[0] = 2 * pc[0] + (k & 1); cc[1] = 2 * pc[1] + ((k >> 1) & 1); cc[2] = 2 * pc[2] + ((k >> 2) & 1);
          for (int g = 0; g < G; g++)
            for (int q = 0; q < 4; q++)
              o->Ul[l][((size_t)g * nc + 8 * oc + k) * 4 + q] = amr_U(o, l - 1)[((size_t)g * o->ncell[l - 1] + p) * 4 + q];
        }
      }
    }
  }
  for (int l = 1; l <= o->n_levels; l++) {
    const int nl = n << l;
    for (int64_t cell = 0; cell < o->ncell[l]; cell++)
      for (int d = 0; d < 3; d++)
        for (int s = -1; s <= 1; s += 2) {
          int c[3] = {o->coord[l][3 * cell], o->coord[l][3 * cell + 1], o->coord[l][3 * cell + 2]};
          c[d] += s;
          if (c[d] < 0 || c[d] >= nl) {
            if (o->bc[2 * d + (s > 0)] != ORC_BC_PERIODIC) continue;
            c[d] = (c[d] + nl) % nl;
          }
          int lf;
          amr_find(o, l, c[0], c[1], c[2], &lf);
          if (lf < l - 1) return ORC_EINVAL;
        }
  }
  o->amr = 1;
  return ORC_OK;
}

/* test hook: the interpolated state (A21) of the virtual level-`level` cell at integer coordinates v[] that
 * lies inside the level-(level-1) leaf `coarse_cell` */
int orc_amr_ghost(orc* o, int level, int group, const int v[3], int64_t coarse_cell, double out[4])
{
  if (!o || !o->amr || level < 1 || level > o->n_levels + 1 || group < 0 || group >= o->ph.G) return ORC_EINVAL;
  if (coarse_cell < 0 || coarse_cell >= o->ncell[level - 1]) return ORC_EINVAL;
  amr_ghost(o, level, group, v, coarse_cell, out);
  return ORC_OK;
}

/* overwrite the radiation of one level and group (tests: random refined states); src is [ncell_l][4] */
int orc_write_U(orc* o, int level, int group, const double* src)
{
  if (!o || level < 0 || level > o->n_levels || group < 0 || group >= o->ph.G || !src) return ORC_EINVAL;
  if (level > 0 && !o->amr) return ORC_EINVAL;
  double* U = amr_U(o, level) + (size_t)group * o->ncell[level] * 4;
  for (int64_t i = 0; i < o->ncell[level] * 4; i++) U[i] = src[i];
  return ORC_OK;
}

/* bottom-up restriction of the radiation after orc_write_U (split cells := children mean) */
int orc_restrict_U(orc* o)
{
  if (!o || !o->amr) return ORC_EINVAL;
  const int G = o->ph.G;
  double v[8];
  for (int l = o->n_levels - 1; l >= 0; l--)
    for (int64_t oc = 0; oc < o->ncell[l + 1] / 8; oc++) {
      int64_t p = o->parent[l + 1][oc];
      for (int g = 0; g < G; g++)
        for (int q = 0; q < 4; q++) {
          for (int k = 0; k < 8; k++) v[k] = o->Ul[l + 1][((size_t)g * o->ncell[l + 1] + 8 * oc + k) * 4 + q];
          amr_U(o, l)[((size_t)g * o->ncell[l] + p) * 4 + q] = mean8(v);
        }
    }
  return ORC_OK;
}
