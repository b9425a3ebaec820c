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
  COSENU_OPT_WENO_EPS = 1, /* epsilon of Eq. (14); default 1e-6; 1e-40 <= eps <= 1e30 (the range the
                              one-division form of the weights supports on every beam, v = 0 included) */
  COSENU_OPT_ADVECT = 2,   /* 0 switches the advection term off (commutator-only runs); default 1 */
  COSENU_OPT_RK_FORM = 3,  /* how the classical RK4 combination is carried between the 4 stage launches
                              (same method, same result up to rounding; differs in HBM traffic per cell-step):
                              0: accumulator array  ACC = u + dt/6 (k1 + 2k2 + 2k3), updated by every stage  (1024 B)
                              1: as 0, but stage 1 does not store ACC; stage 2 rebuilds k1 from (y2 - u) 2/dt  (896 B)
                              2: no accumulator: u+ = (y2 + 2 y3 + y4 - u)/3 + dt/6 k4 from the stage states   (832 B)
                              3: partial sum: stage 2, which holds u, y2 and y3, also stores P = (y2 + 2 y3 - u)/3;
                                 stage 4 reads only P: u+ = P + y4/3 + dt/6 k4                                  (768 B)
                              default 3 */
  COSENU_OPT_STAGE_TIMING = 4, /* 1: bracket every stage launch with CUDA events on the handle's stream
                              (read with cosenu_stage_times); default 0 */
  COSENU_OPT_VARIANT = 5,  /* kernel shape (same arithmetic per cell in all shapes, bit-identical results).
                              FD4+KO: 1: 16 compute warps x 1 row; any other value: 8 compute warps x 2 rows; 16-row tiles always.
                              WENO7, routing per launch by the KIND of the RK stage (the kinds of RK form 0 are FIRST, MID, MID, LAST;
                              form 1: FIRST_LEAN, MID_REBUILD, MID, LAST; form 2: FIRST_LEAN, MID_NOACC, MID_NOACC, LAST_COMB;
                              form 3: FIRST_LEAN, MID_P, MID_NOACC, LAST_P):
                              0 (default): FIRST_LEAN, MID_P, MID_NOACC and LAST_P -- all of form 3, stage 1 of forms 1 and 2, stages 2, 3
                                 of form 2 -- run the marching kernel (csrc/weno_march.cuh: one warp per component marches along z
                                 through a 16-row tile, separate warps combine).  The other kinds run row-block kernels: LAST on 22-row
                                 tiles when those quantise no worse than 16-row tiles over the persistent grid, on 16-row tiles
                                 otherwise; FIRST, MID, MID_REBUILD, LAST_COMB always on 16-row tiles.  One RK step of forms 0-2 can
                                 therefore mix tile heights;
                              4: as 0 for the four marching kinds; every other kind on 16-row tiles (never the tall ones);
                              1: row-block kernels, 16 compute warps x 1 row, 16-row tiles, every kind;
                              2: row-block kernels, every kind; FIRST_LEAN, LAST_P (24 rows, 12 compute warps), MID_NOACC, LAST (22 rows,
                                 11 warps) and MID_P (20 rows, 10 warps) on tall tiles, the rest on 16-row tiles;
                              3: row-block kernels, 8 compute warps x 2 rows on 16-row tiles, every kind */
  COSENU_OPT_GRAPH = 8,    /* 1 (default): cosenu_step(n >= 16) replays a CUDA graph of 8 RK4 steps (32 kernel nodes) captured from the
                              handle's own launches, which removes the per-launch host cost on the small, launch-bound grids;
                              0: always launch kernel by kernel.  Not used on slab handles (their launch parameters change every
                              stage) nor while COSENU_OPT_STAGE_TIMING is on. */
  COSENU_OPT_MAX_CTAS = 9, /* cap of the persistent grid of a stage launch (0, default: one CTA per SM).  With a cap of at most half the SMs
                              the stage kernels of two slab handles driven from two streams are co-resident, which is how the fused
                              halo exchange is exercised on one GPU (tests/test_gpu_slab.py); no other use */
  COSENU_OPT_HALO_TIMEOUT_S = 10, /* z-slab handles: seconds a stage kernel waits for a neighbour's ghost rows before it gives up and
                              flags the run invalid (cosenu_slab_wait_failed); default 4, 0.001 .. 3600.  Raise it where ranks may
                              start a step far apart (a first step after a slow upload on one rank, a debugger, a loaded node). */
  COSENU_OPT_KO_ORDER = 7, /* r of the Kreiss-Oliger operator of Eq. (5): 2 (default; "r = 2 for most numerical
                              experiments"; 5-point, halo 2) or 3 (7-point (eps/64dz) delta^6, halo 3).  FD scheme only;
                              the handle's stream is idle when this is changed. */
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
 * caller-owned cudaStream_t (NULL: the library creates a blocking stream of its own, which orders with the legacy default
 * stream like default-stream work does).  Must be called before init/set_state;
 * if it never is, the library allocates its own workspace with cudaMalloc on first use.
 * The workspace must be plain DEVICE memory (cudaMalloc / a pooled device allocation: cudaPointerGetAttributes type
 * cudaMemoryTypeDevice) of the device the handle was created on: the TMA descriptors and the peer stores of the slab
 * kernels address it directly.  Managed (cudaMallocManaged), pinned-host and pageable memory, and memory of another
 * device, are refused with COSENU_EINVAL. */
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

/* Advance n >= 0 RK4 steps: 4 n kernel launches (kernel by kernel, or as CUDA-graph replays, COSENU_OPT_GRAPH) enqueued on
 * the stream; returns without waiting. */
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

/* Identity of the loaded binary: the first 12 hex digits of the sha1 over the sources it was compiled from (csrc/ in
 * name order, then this header), put in at compile time by paper_2203_12866_b200/build.py ("unknown" for a build made by
 * hand).  bench.py prints it, and quotes an ncu capture under profiles/ only if the capture names the same id. */
const char* cosenu_build_id(void);

/* ===================================================================================================
 * z-slab decomposition over several GPUs (the paper's "future work").
 *
 * The periodic z-grid of nz_global cells is cut into contiguous slabs, one handle (one GPU, one process)
 * per slab.  Everything a cell needs from other cells is (i) all beams v at its own z (the velocity
 * moments of Eq. 3 are local in z, so a slab needs NO reduction collective) and (ii) the stencil halo in z
 * (2 rows for FD4+KO3, 4 for WENO7).  The halo exchange is fused into the stage kernels: the CTA that
 * produces the first / last 4 rows of a stage output also stores them into the neighbouring slab's ghost
 * rows through peer memory (NVLink), then bumps an arrival counter in the neighbour's memory
 * (release, system scope); the neighbour's next stage launch waits on that counter (acquire) only before it
 * loads a tile that touches ghost rows.  Edge tiles are walked first, so the wait is normally over before
 * it starts.  No host synchronisation and no extra launch per stage.
 *
 * Call order on every rank:  create_slab -> [attach(NULL, 0, stream)] -> set options -> slab_export ->
 * (exchange the cosenu_slab_peer_t blobs) -> slab_link -> init / set_state (the LOCAL rows) ->
 * slab_push_ghosts -> (barrier over all ranks) -> slab_ref_sums -> (sum over ranks) -> slab_set_ref_sums ->
 * slab_diag_sums -> (reduce) -> slab_diag_finish(set_reference = 1) -> step ... ; all ranks must advance
 * by the same number of steps.  cosenu_diagnostics is not available on a slab handle (ESTATE): use
 * slab_diag_sums + reduce + slab_diag_finish.
 * =================================================================================================== */

/* What a neighbour needs to reach this slab's ghost rows and counters.  Plain data, safe to send between
 * processes as bytes. */
typedef struct {
  unsigned char ipc_handle[64]; /* cudaIpcMemHandle_t of the allocation that holds the workspace */
  uint64_t ipc_offset;          /* byte offset of the workspace inside that allocation */
  uint64_t dev_base;            /* device address of the workspace in the exporting process */
  int64_t  pid;                 /* exporting process (same pid => linked through dev_base, no IPC) */
  int32_t  device;              /* CUDA device ordinal in the exporting process */
  int32_t  nvp;                 /* row pitch in doubles */
  int64_t  nz_local;            /* rows of the slab */
  int64_t  comp_stride;         /* doubles between two components of a state buffer */
  uint64_t off_buf[4];          /* byte offsets of the four state buffers inside the workspace */
  uint64_t off_ctr;             /* byte offset of the two arrival counters (low ghosts, high ghosts) */
} cosenu_slab_peer_t;

/* A slab that owns rows [z_begin, z_begin + nz_local) of a periodic grid of nz_global cells; dz = L/nz_global.
 * nz_local >= 16.  (nz_local == nz_global, linked to itself, is the single-domain solver again.) */
cosenu_t* cosenu_create_slab(int64_t nz_global, int64_t z_begin, int64_t nz_local, int32_t nv, double L, double dt,
                             double omega, double theta, double mu, int scheme);

/* Allocate the workspace if needed (a slab that is reached over IPC should own its workspace: call
 * cosenu_attach with dev_workspace = NULL to pass only the stream) and describe it. */
int cosenu_slab_export(cosenu_t* h, cosenu_slab_peer_t* out);

/* Connect to the slab below (lo: holds rows just before z_begin, periodically) and above (hi).  Peers of the same
 * process are used through their device addresses; others are mapped with cudaIpcOpenMemHandle. */
int cosenu_slab_link(cosenu_t* h, const cosenu_slab_peer_t* lo, const cosenu_slab_peer_t* hi);

/* After init / set_state: store my edge rows into the neighbours' ghost rows (enqueued on the stream) and wait
 * for the stream.  The caller then synchronises all ranks before the first step. */
int cosenu_slab_push_ghosts(cosenu_t* h);

/* Diagnostics of a decomposed run are sums / maxima over slabs; the caller supplies the reduction.
 *  slab_ref_sums:     out[4][nv] = sum over my rows of |P_nu|, P0_nu, |P_nubar|, P0_nubar per beam
 *  slab_set_ref_sums: the same array summed over all slabs -> the per-beam references of Eq. (22, 23)
 *  slab_diag_sums:    out[10] = 7 sums then 3 maxima over my cells (opaque to the caller: reduce [0..6] by
 *                     sum and [7..9] by max over the slabs)
 *  slab_diag_finish:  global[10] -> *out; set_reference != 0 also stores the t = 0 references (survival
 *                     probability denominators, M0(0)) */
int cosenu_slab_ref_sums(cosenu_t* h, double* out);
int cosenu_slab_set_ref_sums(cosenu_t* h, const double* global_sums);
int cosenu_slab_diag_sums(cosenu_t* h, double* out10);
int cosenu_slab_diag_finish(cosenu_t* h, const double* global10, int set_reference, cosenu_diag_t* out);

/* Several slabs driven by ONE process on ONE stream (e.g. two slabs on one GPU in the tests): advances all of
 * them n steps, stage by stage (every slab's stage k is enqueued before any slab's stage k+1, so no kernel ever
 * waits for a kernel that is queued behind it). */
int cosenu_slab_step_group(cosenu_t** hs, int32_t count, int64_t n);

/* Enqueue ONE RK stage (k = 0..3, in this order; k = 3 completes the step) of a slab.  For drivers that put their own
 * synchronisation between the stages, e.g. several processes sharing one GPU, where a kernel must never have to wait
 * for a kernel of another process: sync + barrier after every stage, so every counter has arrived before the launch. */
int cosenu_slab_stage(cosenu_t* h, int32_t k);

/* 1 if a halo wait of this handle ever timed out (a neighbour did not arrive within COSENU_OPT_HALO_TIMEOUT_S, default 4 s);
 * synchronises. */
int cosenu_slab_wait_failed(cosenu_t* h, int32_t* failed);

/* ===================================================================================================
 * One call that allocates nothing on the device.
 *
 * Who it is for.  Everything above needs a workspace, and somebody has to cudaMalloc it.  Some code that wants a
 * diagnostic of a state cannot do that where it runs:
 *   - a monitor hooked into a production time loop whose process has handed the GPU's memory to a pooling allocator
 *     (PyTorch's caching allocator, RMM, an application arena).  At the 262144 x 512 configuration the solver's own
 *     workspace is 34 GB; a raw cudaMalloc beside the pool either fails for lack of free memory or takes memory the
 *     pool's bookkeeping knows nothing about;
 *   - a monitor that runs while z-slab handles free-run on other streams of the same GPU.  cudaFree (and, depending
 *     on the driver, cudaMalloc) waits for the whole device.  A host thread stuck in that wait cannot enqueue the next
 *     stage of its own slab, the neighbouring slab's kernel spins on the ghost rows that stage would deliver, gives up
 *     after about 4 s, and the run is flagged invalid (cosenu_slab_wait_failed).
 * For them: the per-beam z-sums of the polarisation-vector length and of the trace, the quantities cosenu_slab_ref_sums
 * returns and from which the references |P|_0(v), P0_0(v) of Eq. (22), (23) (Eq. 4)
 * are formed, computed from a state that already sits in device memory.
 *
 *   dev_state  DEVICE pointer, caller-owned, read only: a state in the canonical layout double[8][nz][nv] (dense).
 *   dev_out    DEVICE pointer, caller-owned: double[4][nv], overwritten with
 *              out[0][j] = sum_z |P_nu|(z, v_j),    out[1][j] = sum_z (rho_ee + rho_xx)(z, v_j),
 *              out[2][j], out[3][j] = the same for rhobar;   |P| = sqrt((ee - xx)^2 + 4 (Re ex^2 + Im ex^2)).
 *   cuda_stream  a cudaStream_t (NULL = the legacy default stream).  The two kernel launches are enqueued on it and
 *              the call returns without waiting; dev_out is valid once the stream has reached that point.
 *   Both buffers must belong to the device that is CURRENT when the call is made (managed memory is accepted too).
 *
 * Where the scratch memory comes from.  The per-block partial sums go into a fixed array compiled into the library
 * (148 x 4 x COSENU_STATIC_MAX_NV doubles = 2.3 MiB).  Every GPU on which a process loads this library's device code
 * holds one copy until the process exits, whether or not this call is ever made.
 * Limits: 1 <= nv <= COSENU_STATIC_MAX_NV and 1 <= nz <= 2^40; anything else returns COSENU_EINVAL (the text names
 * the limit) and launches nothing.  Wider v-grids have to use a handle (cosenu_slab_ref_sums).
 * No allocation: the call makes no cudaMalloc, cudaFree, cudaMallocAsync or other allocating CUDA / library call, on
 * the first call or later.  The FIRST call on each device additionally looks up where that device's copy of the array
 * lives (cudaGetSymbolAddress, with that device current, serialised by a mutex) and remembers it; make that first call
 * before any stream capture begins in the process.
 * Sharing: all calls on a device use the SAME array, and it keeps whatever the last call left in it.  Nothing in it
 * has to start at zero (the first launch overwrites every entry the second one reads, for the nv of that call), so
 * successive calls with different nz / nv on one stream are fine.  Two calls that can overlap on the GPU (different
 * streams without an event between them, or two host threads on different streams) race on the array and both results
 * are garbage: order them yourself.  Separate processes have separate copies.
 * Accuracy: not bit-identical to cosenu_slab_ref_sums (which sums the same 148 partials on the host in long double);
 * the two agree to a few ulp of each sum.
 * Errors: returns a COSENU_* code; the text of the calling thread's last failure is at
 * cosenu_beam_sums_static_error() (valid until that thread's next call; empty if none failed).  Host pointers, a
 * buffer of another device, nv or nz out of range -> COSENU_EINVAL; CUDA failures (including: no device) -> COSENU_ECUDA.
 * =================================================================================================== */
#define COSENU_STATIC_MAX_NV 512
int cosenu_beam_sums_static(const double* dev_state, int64_t nz, int32_t nv, double* dev_out, void* cuda_stream);
const char* cosenu_beam_sums_static_error(void);

#ifdef __cplusplus
}
#endif
#endif
