/*
 * cosenu_ref.h -- C ABI of the CPU ORACLE for the COSEnu RK4 hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path under paper_2203_12866_b200/csrc/.
 *
 * What it computes (plain, slow, fp64, in the paper's order and notation):
 *   one classical RK4 step of Eq. (1a,1b) with the Hamiltonian of
 *   Eq. (3a,3b) on a periodic z-grid x bin-centre v-grid,
 *   advection by FD4 + Kreiss-Oliger r=2 (Eq. 5) or by finite volume
 *   with WENO7 (App. A, Algorithm 1).
 *
 * Canonical host layout of a state: double state[8][nz][nv], index (c*nz + iz)*nv + iv,
 *   c0=rho_ee c1=rho_xx c2=Re rho_ex c3=Im rho_ex, c4..c7 the same for rho_bar
 *   (Eq. 2).  rho_bar carries the asymmetry alpha.
 *
 * Parity-pin status: every function below is pinned by
 * tests/test_oracle_*.py except the magnitudes of Figs. 1, 5-11 ("parity unpinned":
 * the paper prints no numbers for them).
 */
#ifndef COSENU_REF_H
#define COSENU_REF_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct cosenu_ref cosenu_ref_t;

enum { COSENU_REF_FD4_KO3 = 0, COSENU_REF_FV_WENO7 = 1 };
enum { COSENU_REF_OK = 0, COSENU_REF_EINVAL = 1, COSENU_REF_ENOMEM = 2, COSENU_REF_ESTATE = 4 };
/* option keys */
enum { COSENU_REF_OPT_EPS_KO = 0,    /* KO strength, default 0.1 */
       COSENU_REF_OPT_WENO_EPS = 1,  /* epsilon of Eq. (14), default 1e-6 */
       COSENU_REF_OPT_ADVECT = 2,    /* test hook: 0 switches the advection term off */
       COSENU_REF_OPT_THREADS = 3,   /* OpenMP threads over z (0 = all) */
       COSENU_REF_OPT_KO_ORDER = 5,  /* r of Eq. (5): 2 (default) or 3 (7-point operator, halo 3) */
       COSENU_REF_OPT_QUADRATURE = 4 }; /* v-grid and rule of the v' integral (set before init / set_state):
                                        0 bin centres + Riemann sum (default);
                                        1 vertex-centred points v_j = -1 + 2j/(nv-1) + trapezoid rule;
                                        2 the same points + Simpson's rule (nv odd) */

typedef struct {
  double t; int64_t step;
  double psurv_nu, psurv_nubar;   /* <rho_ee>(t) of PAPER.md:229, multi-angle reading */
  double dP_max, dP_avg;          /* Eq. (22), Eq. (23) */
  double M0[3], dM0[3];           /* Eq. (19) and its deviation from t=0 */
  double trace_dev_max;           /* max |P0(t) - P0_ref(v)| (Eq. 4 text) */
  double ex_abs_max;              /* max |rho_ex|, |rho_bar_ex| */
} cosenu_ref_diag_t;

cosenu_ref_t* cosenu_ref_create(int64_t nz, int32_t nv, double L, double dt,
                                double omega, double theta, double mu, int scheme);
int  cosenu_ref_set_option(cosenu_ref_t*, int key, double value);
int  cosenu_ref_init(cosenu_ref_t*, uint64_t seed, double sigma_nu, double sigma_nubar,
                     double alpha, double pert_amp, int pert_kind);
int  cosenu_ref_set_state(cosenu_ref_t*, const double* host_state, double t);
int  cosenu_ref_step(cosenu_ref_t*, int64_t n);
int  cosenu_ref_get_state(cosenu_ref_t*, double* host_out);
int  cosenu_ref_diagnostics(cosenu_ref_t*, cosenu_ref_diag_t* out);
void cosenu_ref_destroy(cosenu_ref_t*);
const char* cosenu_ref_last_error(const cosenu_ref_t*);

/* ---- pieces exposed so the pins can test them one by one ---- */
/* k = RHS(y) for an arbitrary state in the canonical layout (does not touch the handle's state) */
int  cosenu_ref_rhs(cosenu_ref_t*, const double* y, double* k);
/* the 6 velocity moments per z: out[6][nz] = M0_Dd, M1_Dd, M0_Dr, M1_Dr, M0_Di, M1_Di */
int  cosenu_ref_moments(cosenu_ref_t*, const double* y, double* out);
/* App. A on one 7-cell stencil f[0..6] = f_{i-3}..f_{i+3}: candidates (A.2), SI (A.3), d_r */
void cosenu_ref_weno7_candidates(const double f[7], double fhat[4]);
void cosenu_ref_weno7_si(const double f[7], double si[4]);
void cosenu_ref_weno7_dr(double d[4]);
/* Algorithm 1: the WENO7 value at i+1/2 */
double cosenu_ref_weno7_face(const double f[7], double eps);

#ifdef __cplusplus
}
#endif
#endif
