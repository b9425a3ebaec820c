/*
 * cosenu.h -- C ABI of cosenu-b200: the RK4 hot path of COSEnu (arXiv 2203.12866) as hand-written
 * sm_100a CUDA.  No torch types, plain pointers and sizes.  Every pointer argument is a HOST pointer
 * unless its name starts with "dev_".
 *
 * What one cosenu_step computes (PAPER.md = /root/reference/PAPER.md of the build):
 *   one classical RK4 step of the two-flavour QKE, Eq. (1a,1b) PAPER.md:41-45,
 *       d_t rho(z,v) = -v d_z rho - i[H, rho],   d_t rhobar = -v d_z rhobar - i[Hbar, rhobar],
 *   with H = H_vac + mu * int dv' (1 - v v') [rho - rhobar^*]  (Eq. 3a),
 *        Hbar = H_vac - mu * int dv' (1 - v v') [rho^* - rhobar] (Eq. 3b),
 *        H_vac = (omega/2) [[-cos2theta, sin2theta],[sin2theta, cos2theta]],
 *   on a periodic z-grid of nz cells (dz = L/nz) times nv bin-centre beams
 *   v_j = -1 + (j + 1/2) 2/nv with the Riemann sum for the v' integral.
 *   The advection term is discretised by
 *     COSENU_FD4_KO3 : 4th-order central differences + Kreiss-Oliger r=2 dissipation,
 *                      Eq. (5) PAPER.md:82-92 (dissipative sign), or
 *     COSENU_FV_WENO7: finite volume, Eq. (7), interface values by the 7th-order
 *                      WENO reconstruction of Eqs. (12)-(14) and App. A / Algorithm 1
 *                       applied to f = v u, upwinded by the sign of v.
 *   Every RK stage is ONE fused kernel launch (moments of the stage input are produced by the
 *   epilogue of the launch that wrote it).
 *
 * Canonical host layout of a state:  double state[8][nz][nv],  index (c*nz + iz)*nv + iv,
 *   c0 = rho_ee, c1 = rho_xx, c2 = Re rho_ex, c3 = Im rho_ex, c4..c7 = the same for rhobar
 *   (Eq. 2).  The stored matrices are the un-normalised ones of Eq. (1)-(3): rhobar
 *   carries the asymmetry alpha.
 *
 * Ownership: the handle is owned by the library (cosenu_destroy frees it and any device memory the
 *   library allocated itself).  Host buffers are caller-owned and never retained.  A workspace passed
 *   to cosenu_attach is caller-owned DEVICE memory and must outlive the handle.
 * Threading: one handle = one GPU (the device current at cosenu_create) = one stream; calls on one
 *   handle must not overlap.
 * Errors: every int function returns a COSENU_* code, never throws or aborts; the text of the last
 *   error is at cosenu_last_error(h) (h = NULL: last failed cosenu_create).  There is NO CPU
 *   fallback: without a usable CUDA device every call fails with COSENU_ECUDA.
 */
#ifndef COSENU_H
#define COSENU_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct cosenu cosenu_t;

enum { COSENU_FD4_KO3 = 0, COSENU_FV_WENO7 = 1 };
enum { COSENU_OK = 0, COSENU_EINVAL = 1, COSENU_ENOMEM = 2, COSENU_ECUDA = 3, COSENU_ESTATE = 4 };

/* option keys of cosenu_set_option */
enum {
  COSENU_OPT_EPS_KO = 0,   /* Kreiss-Oliger strength eps_KO of Eq. (5); default 0.1; >= 0 */
  COSENU_OPT_WENO_EPS = 1, /* epsilon of Eq. (14); default 1e-6; 0 < eps <= 1e30 */
  COSENU_OPT_ADVECT = 2,   /* 0 switches the advection term off (commutator-only runs); default 1 */
  COSENU_OPT_RK_FORM = 3,  /* how the classical RK4 combination is carried between the 4 stage launches
                              (same method, same result up to rounding; differs in HBM traffic per cell-step):
                              0: accumulator array  ACC = u + dt/6 (k1 + 2k2 + 2k3), updated by every stage  (1024 B)
                              1: as 0, but stage 1 does not store ACC; stage 2 rebuilds k1 from (y2 - u) 2/dt  (896 B)
                              2: no accumulator: u+ = (y2 + 2 y3 + y4 - u)/3 + dt/6 k4 from the stage states   (832 B)
                              default 2 */
  COSENU_OPT_STAGE_TIMING = 4, /* 1: bracket every stage launch with CUDA events on the handle's stream
                              (read with cosenu_stage_times); default 0 */
  COSENU_OPT_VARIANT = 5,  /* kernel shape: 0 = 8 compute warps x 2 rows (default), 1 = 16 compute warps x 1 row;
                              same arithmetic per cell, different summation grouping of the moments only */
  COSENU_OPT_QUADRATURE = 6 /* v-grid and rule of the v' integral of Eq. (3); must be set before init / set_state:
                              0: nv bins represented by their centres v_j = -1 + (j + 1/2) 2/nv, Riemann sum (default)
                              1: nv vertex-centred points v_j = -1 + 2 j/(nv-1), trapezoid rule (the FD variant of PAPER.md:82-86)
                              2: the same points, Simpson's rule; needs nv odd, nv >= 3
                              The same weights enter the v-sums of the diagnostics and the normalisation of cosenu_init. */
};

/* Diagnostics.  References are taken when a state is set. */
typedef struct {
  double  t;              /* time */
  int64_t step;           /* steps since init / set_state */
  double  psurv_nu;       /* sum_{z,v} rho_ee(t) / sum_{z,v} rho_ee(0): <rho_ee> of PAPER.md:229, all beams */
  double  psurv_nubar;    /* the same for rhobar_ee */
  double  dP_max;         /* Eq. (22): max_{z,v,species} | |P|/|P|_0(v) - 1 |, |P|_0(v) = z-mean at t = 0 */
  double  dP_avg;         /* Eq. (23): sum_{z,v} | |P_nu| - |P_nu|_0 | / sum_{z,v} |P_nu|_0 */
  double  M0[3];          /* Eq. (19): dz dv sum_{z,v} (2 Re D_ex, -2 Im D_ex, D_ee - D_xx), D = rho - rhobar^* */
  double  dM0[3];         /* M0(t) - M0(0) */
  double  trace_dev_max;  /* max | (rho_ee + rho_xx)(t) - z-mean of (rho_ee + rho_xx)(0) |, both species */
  double  ex_abs_max;     /* max |rho_ex|, |rhobar_ex| */
} cosenu_diag_t;

/* Create a solver on the current CUDA device.  z in [0,L) periodic, dz = L/nz; theta in radians;
 * dt is passed directly (the paper's C_CFL dz / max|v|).  Requires nz >= 16, nv >= 2,
 * L > 0, dt > 0, finite omega/theta/mu, scheme in {0,1}.  Returns NULL on failure. */
cosenu_t* cosenu_create(int64_t nz, int32_t nv, double L, double dt,
                        double omega, double theta, double mu, int scheme);

/* Device memory the solver needs (4 state copies in the device layout + moment and scratch arrays). */
size_t cosenu_workspace_bytes(const cosenu_t* h);

/* Optional: use caller-owned device memory (>= cosenu_workspace_bytes, 256-byte aligned) and a
 * caller-owned cudaStream_t (NULL = legacy default stream).  Must be called before init/set_state;
 * if it never is, the library allocates its own workspace with cudaMalloc on first use. */
int cosenu_attach(cosenu_t* h, void* dev_workspace, size_t bytes, void* cuda_stream);

int cosenu_set_option(cosenu_t* h, int key, double value);

/* Seeded initial state (angular distributions of Eq. (20), discretely normalised,
 * rhobar scaled by alpha; off-diagonal seed of amplitude pert_amp):
 *   pert_kind 0: rho_ex = pert_amp g_j exp(i phi_z), phi_z = 2 pi u_z, u_z the splitmix64(seed) stream
 *             1: band-limited: 16 lowest Fourier modes with seeded phases
 *             2: Eq. (21): eps(z) = pert_amp exp(-(z - L/2)^2 / 50), pure state
 * The state is built on the host and uploaded (t = 0). */
int cosenu_init(cosenu_t* h, uint64_t seed, double sigma_nu, double sigma_nubar, double alpha,
                double pert_amp, int pert_kind);

/* Upload an arbitrary state (canonical host layout) and set the time. */
int cosenu_set_state(cosenu_t* h, const double* host_state, double t);

/* Advance n >= 0 RK4 steps: 4 n kernel launches enqueued on the stream, returns without waiting. */
int cosenu_step(cosenu_t* h, int64_t n);

/* Wait for the stream and copy the state to host_out (canonical host layout, 8*nz*nv doubles). */
int cosenu_get_state(cosenu_t* h, double* host_out);

/* Copy the 6 velocity moments of the current state, double out[6][nz]:
 * M0_Dd, M1_Dd, M0_Dr, M1_Dr, M0_Di, M1_Di with M^k_X(z) = dv sum_j v_j^k X(z,j),
 * Dd = (rho_ee-rho_xx)-(rhobar_ee-rhobar_xx), Dr = Re(rho_ex - rhobar_ex^*), Di = Im(same). */
int cosenu_get_moments(cosenu_t* h, double* host_out);

/* Reduce the diagnostics on the device, wait, and fill *out. */
int cosenu_diagnostics(cosenu_t* h, cosenu_diag_t* out);

/* Wait for all work enqueued on the handle's stream. */
int cosenu_sync(cosenu_t* h);

/* Number of kernel launches issued through this handle so far (for the bench's gpu_launches). */
int64_t cosenu_launch_count(const cosenu_t* h);

/* With COSENU_OPT_STAGE_TIMING on: waits for the stream, then returns the device time of the stage
 * kernels, summed per RK stage over all steps run since the option was switched on (or since the last
 * call): ms_sum[4] in milliseconds, *launches_per_stage = number of steps summed. */
int cosenu_stage_times(cosenu_t* h, double* ms_sum, int64_t* launches_per_stage);

void cosenu_destroy(cosenu_t* h);
const char* cosenu_last_error(const cosenu_t* h);

#ifdef __cplusplus
}
#endif
#endif
