// cosenu_api.cu -- the C ABI of include/cosenu.h: handle, workspace, TMA descriptors, launches.
// Host logic only; every step of the path runs in the kernels of stage_kernels.cuh / aux_kernels.cuh.
#include "../../include/cosenu.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <unistd.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <set>
#include <string>
#include <vector>

#include "aux_kernels.cuh"
#include "stage_kernels.cuh"
#include "weno_march.cuh"

using namespace cosenu_dev;

namespace {

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// tile shapes: TZ rows per tile, NSEG compute warps (S = TZ/NSEG rows each),
// NY / NUA ring depths of the stage-input and of the u0/acc shared-memory slots.  `variant` picks a row.
constexpr int TZ_ALL = 16;
constexpr int TZ_WENO1 = 24;   // WENO7, kinds that stage one array: 12 compute warps x 2 rows
constexpr int TZ_WENO3 = 20;   // ... 10 compute warps x 2 rows: stage 2 of RK form 3, which stages two arrays
constexpr int TZ_WENO2 = 22;   // ... 11 compute warps x 2 rows (the kind that needs more than 128 registers)
constexpr int DIAG_BLOCKS = 592, DIAG_THREADS = 256, REF_BLOCKS = 148;

std::string g_create_err;

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace

struct cosenu {
  int64_t nz; int32_t nv; int nvp;
  double L, dt, omega, theta, mu; int scheme;
  double eps_ko = 0.1, weno_eps = 1e-6;
  int advect = 1, rk_form = 3, stage_timing = 0;   // rk_form: 0 accumulator, 1 lean accumulator, 2 accumulator-free, 3 partial sum
  int quad = 0;          // COSENU_OPT_QUADRATURE
  int ko_r = 2;          // COSENU_OPT_KO_ORDER: r of Eq. (5)
  double dz, dv, voff = 0.5;   // v_j = -1 + (j + voff) dv
  int device = 0;
  int variant = 0;       // kernel shape variant (COSENU_OPT_VARIANT)
  int num_sms = 148;
  int max_ctas = 0;      // COSENU_OPT_MAX_CTAS: cap of the persistent grid of a stage launch (0: one CTA per SM)
  double halo_timeout_s = 4.0;   // COSENU_OPT_HALO_TIMEOUT_S: how long a slab's halo wait may last

  // workspace
  void* ws = nullptr; size_t ws_bytes = 0; bool ws_owned = false;
  cudaStream_t stream = nullptr;
  double *U = nullptr, *Y1 = nullptr, *Y2 = nullptr, *ACC = nullptr;
  double* M[2] = {nullptr, nullptr};
  double *d_pref = nullptr, *d_p0ref = nullptr, *d_refpart = nullptr, *d_diagpart = nullptr;
  int64_t comp_stride = 0; size_t state_elems = 0;
  int mcur = 0;  // M[mcur] holds the moments of U
  // tensor maps per tile height (index 0: TZ = 16; WENO7 only: 1: TZ = 24, 2: TZ = 22, 3: TZ = 20) and per state buffer
  // (0 U, 1 Y1, 2 Y2, 3 ACC)
  CUtensorMap tm[4][4];   // stage-input boxes [8][TZ+2H][32] over the ghosted rows
  CUtensorMap tp[4][4];   // rows 0..nz-1 only, boxes [8][TZ][32]: u0 / acc loads, output stores
  bool maps_ready = false;

  bool have_state = false;
  double t = 0; int64_t step = 0;
  int64_t launches = 0;
  double sum_ee0[2] = {0, 0}, M0_init[3] = {0, 0, 0}, pref_sum_nu = 0;

  // stage timing
  std::vector<cudaEvent_t> ev_pool; size_t ev_used = 0;
  double stage_ms[4] = {0, 0, 0, 0}; int64_t stage_n = 0;

  std::set<const void*> configured;   // stage kernels whose shared-memory attribute is set on this device
  bool dry_run = false;               // launch_one only sets the kernel attributes (before a stream capture)

  // CUDA graph of GRAPH_STEPS RK4 steps (4 GRAPH_STEPS kernel nodes): replayed by cosenu_step when the launch
  // parameters repeat from step to step (single domain, no per-stage events)
  bool stream_owned = false;
  int use_graph = 1;
  cudaGraphExec_t gexec = nullptr;

  // z-slab decomposition (cosenu_create_slab): this handle owns rows [z_begin, z_begin + nz) of nz_global
  bool slab = false, linked = false, ghosts_pushed = false;
  int64_t nz_global = 0, z_begin = 0;
  unsigned long long* d_ctr = nullptr;   // my arrival counters: [0] low ghost rows, [1] high ghost rows
  int* d_err = nullptr;                  // halo wait gave up
  double* peer_buf[2][4] = {{nullptr, nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr, nullptr}};  // [lo|hi][U,Y1,Y2,ACC]
  int64_t peer_stride[2] = {0, 0}, peer_nz[2] = {0, 0};
  unsigned long long* peer_ctr[2] = {nullptr, nullptr};   // lo peer's HIGH counter, hi peer's LOW counter
  void* ipc_mapped[2] = {nullptr, nullptr};               // bases returned by cudaIpcOpenMemHandle (closed in destroy)
  unsigned long long epoch = 0;                           // stage launches since the link

  std::string err;
};

namespace {

int fail(cosenu* h, int code, const std::string& msg) {
  if (h) h->err = msg; else g_create_err = msg;
  return code;
}
int cuda_fail(cosenu* h, cudaError_t e, const char* what) {
  return fail(h, COSENU_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
// every entry point that touches CUDA runs on the handle's device and leaves the caller's current device as it found it
// (active = false: an entry point that turns out not to touch CUDA makes no runtime call at all -- cudaGetDevice alone would
// create a primary context on whatever device the caller has current)
struct DeviceGuard {
  int prev = -1; bool changed = false;
  explicit DeviceGuard(int dev, bool active = true) {
    if (active && cudaGetDevice(&prev) == cudaSuccess && prev != dev) changed = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() { if (changed) cudaSetDevice(prev); }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define CK(call)                                                  \
  do {                                                            \
    cudaError_t e_ = (call);                                      \
    if (e_ != cudaSuccess) return cuda_fail(h, e_, #call);        \
  } while (0)

// z-slab: a halo wait that gave up (a neighbour that never delivered its rows) leaves stale ghost rows behind: every call
// that hands results to the caller reports it.  The stream is idle here (the callers have just synchronised it).
// The flag is read on the handle's OWN stream: a plain cudaMemcpy runs on the legacy default stream and would first wait
// for every blocking stream of the device -- i.e. for another slab's queued stages, which in turn spin on the stage this
// thread has not launched yet, until their halo wait times out.
int halo_check(cosenu* h, const char* who) {
  if (!h->slab || !h->maps_ready) return COSENU_OK;
  int v = 0;
  CK(cudaMemcpyAsync(&v, h->d_err, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  if (v) return fail(h, COSENU_ESTATE, std::string(who) + ": a halo wait timed out (a neighbouring slab never delivered its ghost rows); the state is invalid");
  return COSENU_OK;
}

size_t workspace_layout(const cosenu* h, size_t off[11]) {
  const size_t st = align_up(sizeof(double) * 8 * (size_t)(h->nz + 2 * G) * h->nvp, 256);
  const size_t mo = align_up(sizeof(double) * 6 * (size_t)h->nz, 256);
  const size_t rf = align_up(sizeof(double) * 2 * (size_t)h->nv, 256);
  const size_t rp = align_up(sizeof(double) * REF_BLOCKS * 4 * (size_t)h->nv, 256);
  const size_t dp = align_up(sizeof(double) * DIAG_BLOCKS * DIAG_NVAL, 256);
  size_t o = 0;
  off[0] = o; o += st;  // U
  off[1] = o; o += st;  // Y1
  off[2] = o; o += st;  // Y2
  off[3] = o; o += st;  // ACC
  off[4] = o; o += mo;  // M[0]
  off[5] = o; o += mo;  // M[1]
  off[6] = o; o += rf;  // pref
  off[7] = o; o += rf;  // p0ref
  off[8] = o; o += rp;  // ref partials
  off[9] = o; o += dp;  // diag partials
  off[10] = o; o += 256; // slab arrival counters (2 x u64) and the wait-failed flag (int, at +64)
  return o;
}

// with_ghosts: the view covers device rows 0..nz+2G-1 (stencil input); otherwise rows G..G+nz-1 (z = 0..nz-1),
// so that out-of-range rows of a ragged last tile are clipped by the TMA store instead of hitting ghost rows
int make_map(cosenu* h, PFN_encodeTiled enc, CUtensorMap* map, double* base, int rows_box, bool with_ghosts) {
  if (!with_ghosts) base += (size_t)G * h->nvp;
  const cuuint64_t gdim[3] = {(cuuint64_t)h->nv, (cuuint64_t)(with_ghosts ? h->nz + 2 * G : h->nz), 8};
  const cuuint64_t gstr[2] = {(cuuint64_t)h->nvp * 8, (cuuint64_t)h->comp_stride * 8};
  const cuuint32_t box[3] = {(cuuint32_t)VC, (cuuint32_t)rows_box, 8};
  const cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(h, COSENU_ECUDA, "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")");
  return COSENU_OK;
}

int make_maps(cosenu* h);

int ensure_workspace(cosenu* h) {
  if (h->maps_ready) return COSENU_OK;
  CK(cudaSetDevice(h->device));
  if (!h->stream) {
    // no caller stream: a BLOCKING stream of our own.  It orders with the legacy default stream exactly as
    // default-stream work would (implicit synchronisation both ways), and unlike the legacy stream it can be captured.
    CK(cudaStreamCreate(&h->stream));
    h->stream_owned = true;
  }
  size_t off[11];
  const size_t need = workspace_layout(h, off);
  if (!h->ws) {
    cudaError_t e = cudaMalloc(&h->ws, need);
    if (e != cudaSuccess) { h->ws = nullptr; return fail(h, e == cudaErrorMemoryAllocation ? COSENU_ENOMEM : COSENU_ECUDA,
                                                        std::string("cudaMalloc workspace: ") + cudaGetErrorString(e)); }
    h->ws_bytes = need; h->ws_owned = true;
  }
  char* b = static_cast<char*>(h->ws);
  h->U = (double*)(b + off[0]); h->Y1 = (double*)(b + off[1]); h->Y2 = (double*)(b + off[2]); h->ACC = (double*)(b + off[3]);
  h->M[0] = (double*)(b + off[4]); h->M[1] = (double*)(b + off[5]);
  h->d_pref = (double*)(b + off[6]); h->d_p0ref = (double*)(b + off[7]);
  h->d_refpart = (double*)(b + off[8]); h->d_diagpart = (double*)(b + off[9]);
  h->d_ctr = (unsigned long long*)(b + off[10]); h->d_err = (int*)(b + off[10] + 64);
  CK(cudaMemsetAsync(h->ws, 0, need, h->stream));

  int rc = make_maps(h);
  if (rc) return rc;
  h->maps_ready = true;
  return COSENU_OK;
}

// halo of the stage-input boxes: 2 rows for FD4 + KO r = 2, 3 for KO r = 3, 4 for WENO7
int make_maps(cosenu* h) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qr;
  CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr));
  if (!fn || qr != cudaDriverEntryPointSuccess) return fail(h, COSENU_ECUDA, "cuTensorMapEncodeTiled not available in this driver");
  PFN_encodeTiled enc = reinterpret_cast<PFN_encodeTiled>(fn);
  const int halo = h->scheme == COSENU_FD4_KO3 ? h->ko_r : 4;
  double* bufs[4] = {h->U, h->Y1, h->Y2, h->ACC};
  const int tzs[4] = {TZ_ALL, TZ_WENO1, TZ_WENO2, TZ_WENO3};
  for (int t = 0; t < 4; ++t) {
    if (t >= 1 && h->scheme != COSENU_FV_WENO7) continue;
    for (int b = 0; b < 4; ++b) {
      int rc;
      if ((rc = make_map(h, enc, &h->tm[t][b], bufs[b], tzs[t] + 2 * halo, true))) return rc;
      if ((rc = make_map(h, enc, &h->tp[t][b], bufs[b], tzs[t], false))) return rc;
    }
  }
  return COSENU_OK;
}

// persistent grid of a stage launch: one CTA per SM, fewer when there are fewer tiles or the caller caps it (COSENU_OPT_MAX_CTAS)
unsigned grid_size(const cosenu* h, long long ntiles) {
  long long g = ntiles < h->num_sms ? ntiles : h->num_sms;
  if (h->max_ctas > 0 && g > h->max_ctas) g = h->max_ctas;
  return (unsigned)g;
}

template <int SCHEME, int KIND, int TZ, int NSEG, int NY, int NUA>
int launch_one(cosenu* h, int in_buf, int out_buf, int a1_buf, int a2_buf, const StageParams& p0) {
  constexpr int T = TZ == TZ_ALL ? 0 : (TZ == TZ_WENO1 ? 1 : (TZ == TZ_WENO2 ? 2 : 3));
  const CUtensorMap &map = h->tm[T][in_buf], &omap = h->tp[T][out_buf], &a1 = h->tp[T][a1_buf], &a2 = h->tp[T][a2_buf];
  auto kern = stage_kernel<SCHEME, KIND, TZ, NSEG, NY, NUA>;
  constexpr size_t smem = StageSmem<SCHEME, KIND, TZ, NSEG, NY, NUA>::bytes;
  static_assert(smem <= 232448, "over the 227 KB shared-memory limit of a CTA");
  // the opt-in to > 48 KB of dynamic shared memory is per function and per device: remember it per handle
  const void* key = reinterpret_cast<const void*>(kern);
  if (h->configured.find(key) == h->configured.end()) {
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    h->configured.insert(key);
  }
  if (h->dry_run) return COSENU_OK;
  const long long ntiles = (h->nz + TZ - 1) / TZ;
  const unsigned grid = grid_size(h, ntiles);   // persistent: one CTA per SM
  StageParams p = p0;
  if (h->slab) p.tile_shift = ntiles >= 3 ? ntiles - 2 : 0;   // walk the (up to two) high edge tiles, then tile 0, first
  kern<<<grid, NSEG * 32 + 32, smem, h->stream>>>(map, h->tp[T][0], a1, a2, omap, p);
  CK(cudaGetLastError());
  h->launches++;
  return COSENU_OK;
}

// WENO7, partial-sum RK carrier: the role-specialised marching kernel (weno_march.cuh) on 16-row tiles
template <int KIND>
int launch_march(cosenu* h, int in_buf, int out_buf, int acc_buf, const StageParams& p0) {
  auto kern = weno_march_kernel<KIND>;
  constexpr size_t smem = MarchSmem::bytes;
  static_assert(smem <= 232448, "over the 227 KB shared-memory limit of a CTA");
  const void* key = reinterpret_cast<const void*>(kern);
  if (h->configured.find(key) == h->configured.end()) {
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    h->configured.insert(key);
  }
  if (h->dry_run) return COSENU_OK;
  const long long ntiles = (h->nz + MTZ - 1) / MTZ;
  const unsigned grid = grid_size(h, ntiles);   // persistent: one CTA per SM
  StageParams p = p0;
  if (h->slab) p.tile_shift = ntiles >= 3 ? ntiles - 2 : 0;
  kern<<<grid, MARCH_THREADS, smem, h->stream>>>(h->tm[0][in_buf], h->tp[0][0], h->tp[0][acc_buf], h->tp[0][out_buf], p);
  CK(cudaGetLastError());
  h->launches++;
  return COSENU_OK;
}

template <int SCHEME, int TZ, int NSEG, int NY, int NUA, int NUA1 = NUA>   // NUA1: ring depth of the kinds that stage ONE array
int launch_kind(cosenu* h, int kind, int map, int omap, int a1, int a2, const StageParams& p) {
  // kinds that stage ONE array (they also fit tiles of TZ_WENO1 rows)
  switch (kind) {
    // stage 1 of the lean forms loads nothing but the stage input.  The DMA warp issues the store of item n - NUA before it
    // goes on to the load of item n + 1, so its look-ahead is min(NY, NUA) items: 3 + 3 slots beat 4 + 2 (FD, HBM-bound)
    case FIRST_LEAN: return launch_one<SCHEME, FIRST_LEAN, TZ, NSEG, (SCHEME == 1 ? NY : 3), (SCHEME == 0 ? 3 : NUA1)>(h, map, omap, a1, a2, p);   // KO r = 3 (halo 3): 3 + 2 is all that fits
    case LAST: return launch_one<SCHEME, LAST, TZ, NSEG, NY, NUA1>(h, map, omap, a1, a2, p);
    case MID_NOACC: return launch_one<SCHEME, MID_NOACC, TZ, NSEG, NY, NUA1>(h, map, omap, a1, a2, p);
    case LAST_P: return launch_one<SCHEME, LAST_P, TZ, NSEG, NY, NUA1>(h, map, omap, a1, a2, p);
    default: break;
  }
  if constexpr (TZ == TZ_ALL) {   // two or three staged arrays
    switch (kind) {
      case FIRST: return launch_one<SCHEME, FIRST, TZ, NSEG, NY, NUA>(h, map, omap, a1, a2, p);
      case MID: return launch_one<SCHEME, MID, TZ, NSEG, NY, NUA>(h, map, omap, a1, a2, p);
      case MID_REBUILD: return launch_one<SCHEME, MID_REBUILD, TZ, NSEG, NY, NUA>(h, map, omap, a1, a2, p);
      case MID_P: return launch_one<SCHEME, MID_P, TZ, NSEG, NY, NUA>(h, map, omap, a1, a2, p);
      case LAST_COMB: return launch_one<SCHEME, LAST_COMB, TZ, NSEG, NY, 1>(h, map, omap, a1, a2, p);   // 3 staged arrays: one slot
      default: break;
    }
  }
  return fail(h, COSENU_EINVAL, "launch_kind: no kernel for this stage kind and tile height");
}

int launch_stage(cosenu* h, int kind, int map, int omap, int a1, int a2, const StageParams& p) {
  if (h->scheme == COSENU_FD4_KO3 && h->ko_r == 3) {   // FD4 + Kreiss-Oliger r = 3: halo 3
    if (h->variant == 1) return launch_kind<2, TZ_ALL, 16, 2, 2>(h, kind, map, omap, a1, a2, p);
    return launch_kind<2, TZ_ALL, 8, 2, 2>(h, kind, map, omap, a1, a2, p);
  }
  if (h->scheme == COSENU_FD4_KO3) {
    if (h->variant == 1) return launch_kind<0, TZ_ALL, 16, 2, 2>(h, kind, map, omap, a1, a2, p);
    return launch_kind<0, TZ_ALL, 8, 2, 2>(h, kind, map, omap, a1, a2, p);
  }
  if (h->variant == 1) return launch_kind<1, TZ_ALL, 16, 2, 1>(h, kind, map, omap, a1, a2, p);
  if (h->variant == 0 || h->variant == 4) {   // default: the marching kernel (weno_march.cuh) for the kinds of the partial-sum RK carrier
    switch (kind) {
      case FIRST_LEAN: return launch_march<FIRST_LEAN>(h, map, omap, a1, p);
      case MID_P: return launch_march<MID_P>(h, map, omap, a1, p);
      case MID_NOACC: return launch_march<MID_NOACC>(h, map, omap, a1, p);
      case LAST_P: return launch_march<LAST_P>(h, map, omap, a1, p);
      default: break;   // the other RK carriers run the row-block kernels below
    }
  }
  // the kinds that stage one array leave room for taller tiles and more compute warps, unless the coarser tiles quantise
  // worse over the persistent grid (rows walked by the busiest CTA): e.g. nz = 32768 is 13.8 waves of 16-row tiles but
  // 9.2 waves of 24-row tiles
  const long long w16 = ((h->nz + TZ_ALL - 1) / TZ_ALL + h->num_sms - 1) / h->num_sms * TZ_ALL;
  const long long w24 = ((h->nz + TZ_WENO1 - 1) / TZ_WENO1 + h->num_sms - 1) / h->num_sms * TZ_WENO1;
  const bool tz24 = h->variant == 2 || (h->variant == 0 && 0.93 * (double)w24 <= (double)w16);   // variant 3: never
  if (tz24) {
    // Three compute warps per scheduler instead of two hide the fp64 latencies much better (FP64 pipe 81 % busy instead of
    // 71 %): 12 warps x 2 rows on 24-row tiles.  13 warps cap the kernel at 128 registers, which MID_NOACC does not fit
    // without spilling in its hot loop: that kind runs 11 warps x 2 rows on 22-row tiles (12 warps in all, 166 registers).
    switch (kind) {
      case FIRST_LEAN: return launch_one<1, FIRST_LEAN, TZ_WENO1, 12, 2, 1>(h, map, omap, a1, a2, p);
      case LAST_P: return launch_one<1, LAST_P, TZ_WENO1, 12, 2, 1>(h, map, omap, a1, a2, p);
      case MID_NOACC: return launch_one<1, MID_NOACC, TZ_WENO2, 11, 2, 1>(h, map, omap, a1, a2, p);
      case LAST: return launch_one<1, LAST, TZ_WENO2, 11, 2, 1>(h, map, omap, a1, a2, p);
      case MID_P: return launch_one<1, MID_P, TZ_WENO3, 10, 2, 1>(h, map, omap, a1, a2, p);   // two staged arrays: 20 rows is what fits
      default: break;
    }
  }
  return launch_kind<1, TZ_ALL, 8, 2, 1>(h, kind, map, omap, a1, a2, p);
}

StageParams base_params(const cosenu* h) {
  StageParams p;
  std::memset(&p, 0, sizeof(p));
  p.nz = h->nz; p.nv = h->nv; p.nvp = h->nvp; p.comp_stride = h->comp_stride;
  p.mu = h->mu;
  p.A0 = -h->omega * std::cos(2.0 * h->theta);
  p.Br0 = 0.5 * h->omega * std::sin(2.0 * h->theta);
  p.dv = h->dv; p.voff = h->voff; p.quad = h->quad;
  const double sw = h->advect ? 1.0 : 0.0;
  p.cadv = sw * (-1.0 / (12.0 * h->dz));
  p.cko = h->ko_r == 3 ? sw * (h->eps_ko / (64.0 * h->dz)) : sw * (-h->eps_ko / (16.0 * h->dz));
  p.ninv_dz = sw * (-1.0 / h->dz);
  p.weno_eps = h->weno_eps;
  return p;
}

cudaEvent_t next_event(cosenu* h) {
  if (h->ev_used == h->ev_pool.size()) {
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
    h->ev_pool.push_back(e);
  }
  return h->ev_pool[h->ev_used++];
}

int drain_events(cosenu* h) {
  if (h->ev_used == 0) return COSENU_OK;
  CK(cudaStreamSynchronize(h->stream));
  for (size_t s = 0; s + 5 <= h->ev_used; s += 5) {
    for (int k = 0; k < 4; ++k) {
      float ms = 0;
      CK(cudaEventElapsedTime(&ms, h->ev_pool[s + k], h->ev_pool[s + k + 1]));
      h->stage_ms[k] += ms;
    }
    h->stage_n++;
  }
  h->ev_used = 0;
  return COSENU_OK;
}

// y_out = state buffer `which` (0 U, 1 Y1, 2 Y2, 3 ACC) and where the ghost copies of its edge rows go:
// my own periodic ghost rows, or (z-slab) the neighbouring slabs' ghost rows of the same buffer + the arrival counters
void set_output(cosenu* h, StageParams& p, int which) {
  double* bufs[4] = {h->U, h->Y1, h->Y2, h->ACC};
  p.y_out = bufs[which];
  if (!h->slab) {
    p.ghost_lo_dst = p.y_out + (size_t)(h->nz + G) * h->nvp;   // rows 0..G-1 -> device rows nz+G.. (high ghosts)
    p.ghost_hi_dst = p.y_out;                                    // rows nz-G..nz-1 -> device rows 0..G-1 (low ghosts)
    p.ghost_lo_stride = p.ghost_hi_stride = h->comp_stride;
    return;
  }
  // my low rows are the HIGH ghost rows of the slab below; my high rows are the LOW ghost rows of the slab above
  p.ghost_lo_dst = h->peer_buf[0][which] + (size_t)(h->peer_nz[0] + G) * h->nvp;
  p.ghost_lo_stride = h->peer_stride[0];
  p.ghost_hi_dst = h->peer_buf[1][which];
  p.ghost_hi_stride = h->peer_stride[1];
  p.sig_lo = h->peer_ctr[0];
  p.sig_hi = h->peer_ctr[1];
  p.wait_lo = h->d_ctr;
  p.wait_hi = h->d_ctr + 1;
  p.wait_val = (unsigned long long)G * h->epoch;   // G rows per edge per stage launch so far
  p.err_flag = h->d_err;
  p.wait_timeout_ns = (unsigned long long)(h->halo_timeout_s * 1e9);
}

// RK stage k (0..3) of the classical RK4 step = ONE fused launch.  Buffers: U -> Y1 -> Y2 -> (Y1 | ACC) -> U; in the
// accumulator-free form the fourth state buffer (ACC) holds Y4, so that Y2 (in Y1) and Y3 (in Y2) are still there for
// the final combination.  Moments ping-pong between M[mcur] (of U) and M[mcur ^ 1].
int rk_stage(cosenu* h, int k) {
  const double dt = h->dt;
  StageParams p = base_params(h);
  double* Min = h->M[h->mcur];
  double* Mout = h->M[h->mcur ^ 1];
  const int form = h->rk_form;
  int rc = COSENU_OK;
  switch (k) {
    case 0:   // k1 = RHS(U); Y1 = U + dt/2 k1; [ACC = U + dt/6 k1]
      set_output(h, p, 1); p.acc_out = h->ACC; p.mom_in = Min; p.mom_out = Mout;
      p.cy = 0.5 * dt; p.ca = dt / 6.0;
      rc = launch_stage(h, form == 0 ? FIRST : FIRST_LEAN, 0, 1, 3, 3, p);
      break;
    case 1:   // k2 = RHS(Y1); Y2 = U + dt/2 k2; [ACC += dt/3 k2]
      set_output(h, p, 2); p.acc_out = h->ACC; p.mom_in = Mout; p.mom_out = Min;
      p.cy = 0.5 * dt; p.ca = dt / 3.0;
      rc = launch_stage(h, form == 0 ? MID : (form == 1 ? MID_REBUILD : (form == 3 ? MID_P : MID_NOACC)), 1, 2, 3, 3, p);   // form 3: the "accumulator" written here is P = (Y2 + 2 Y3 - U)/3
      break;
    case 2:   // k3 = RHS(Y2); Y4 = U + dt k3 (into Y1, or into ACC in the accumulator-free form); [ACC += dt/3 k3]
      set_output(h, p, form == 2 ? 3 : 1); p.acc_out = h->ACC; p.mom_in = Min; p.mom_out = Mout;
      p.cy = dt; p.ca = dt / 3.0;
      rc = launch_stage(h, (form == 2 || form == 3) ? MID_NOACC : MID, 2, form == 2 ? 3 : 1, 3, 3, p);
      break;
    default:  // k4 = RHS(Y4); U = ACC + dt/6 k4   or   U = (Y2 + 2 Y3 + Y4 - U)/3 + dt/6 k4
      set_output(h, p, 0); p.acc_out = nullptr; p.mom_in = Mout; p.mom_out = Min;
      p.cy = dt / 6.0; p.ca = 0.0;
      if (form == 2) rc = launch_stage(h, LAST_COMB, 3, 0, 1, 2, p);
      else rc = launch_stage(h, form == 3 ? LAST_P : LAST, 1, 0, 3, 3, p);
      break;
  }
  if (rc == COSENU_OK && !h->dry_run) h->epoch++;
  return rc;
}

// one classical RK4 step = 4 fused stage launches (the moments of the new U end up in M[mcur] again)
int one_step(cosenu* h) {
  const bool tm = h->stage_timing != 0;
  int rc;
  cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  if (tm) {
    if (h->ev_used + 5 > 5 * 4096) { if ((rc = drain_events(h))) return rc; }
    for (int k = 0; k < 5; ++k) if (!(ev[k] = next_event(h))) return fail(h, COSENU_ECUDA, "cudaEventCreate failed");
    CK(cudaEventRecord(ev[0], h->stream));
  }
  for (int k = 0; k < 4; ++k) {
    if ((rc = rk_stage(h, k))) return rc;
    if (tm) CK(cudaEventRecord(ev[k + 1], h->stream));
  }
  h->t += h->dt; h->step += 1;
  return COSENU_OK;
}

// ---- diagnostics in four pieces, so that a decomposed run can put its reduction between them
// (1) per-beam sums over my rows of |P_nu|, P0_nu, |P_nubar|, P0_nubar: out[4][nv]
int ref_sums(cosenu* h, double* out) {
  diag_ref_kernel<<<REF_BLOCKS, DIAG_REF_ROWS * DIAG_REF_LANES, 0, h->stream>>>(h->U, h->d_refpart, h->nz, h->nv, h->nvp, h->comp_stride, G);
  CK(cudaGetLastError());
  h->launches++;
  std::vector<double> part((size_t)REF_BLOCKS * 4 * h->nv);
  CK(cudaMemcpyAsync(part.data(), h->d_refpart, sizeof(double) * part.size(), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  for (int m = 0; m < 4; ++m)
    for (int j = 0; j < h->nv; ++j) {
      long double a = 0;
      for (int b = 0; b < REF_BLOCKS; ++b) a += part[((size_t)b * 4 + m) * h->nv + j];
      out[(size_t)m * h->nv + j] = (double)a;
    }
  return COSENU_OK;
}
// (2) the same sums over the whole grid -> references |P|_0(v), P0_0(v) = z-means at t = 0 (Eq. 22, 23)
int set_ref_sums(cosenu* h, const double* sums) {
  const int nv = h->nv;
  const double nzg = (double)(h->slab ? h->nz_global : h->nz);
  std::vector<double> pref(2 * (size_t)nv), p0ref(2 * (size_t)nv);
  long double prsum = 0;
  for (int j = 0; j < nv; ++j) {
    pref[j] = sums[j] / nzg; p0ref[j] = sums[(size_t)nv + j] / nzg;
    pref[nv + j] = sums[2 * (size_t)nv + j] / nzg; p0ref[nv + j] = sums[3 * (size_t)nv + j] / nzg;
    prsum += (long double)quad_weight(j, nv, h->quad) * pref[j];
  }
  h->pref_sum_nu = (double)(prsum * nzg);
  CK(cudaMemcpyAsync(h->d_pref, pref.data(), sizeof(double) * pref.size(), cudaMemcpyHostToDevice, h->stream));
  CK(cudaMemcpyAsync(h->d_p0ref, p0ref.data(), sizeof(double) * p0ref.size(), cudaMemcpyHostToDevice, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return COSENU_OK;
}
// (3) sums [0..6] and maxima [7..9] over my cells
int diag_sums(cosenu* h, double* out10) {
  diag_kernel<<<DIAG_BLOCKS, DIAG_THREADS, 0, h->stream>>>(h->U, h->d_pref, h->d_p0ref, h->d_diagpart, h->nz, h->nv,
                                                           h->nvp, h->comp_stride, G, h->quad);
  CK(cudaGetLastError());
  h->launches++;
  std::vector<double> part((size_t)DIAG_BLOCKS * DIAG_NVAL);
  CK(cudaMemcpyAsync(part.data(), h->d_diagpart, sizeof(double) * part.size(), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  long double s[DIAG_NSUM];
  for (int k = 0; k < DIAG_NSUM; ++k) s[k] = 0;
  for (int k = 0; k < DIAG_NMAX; ++k) out10[DIAG_NSUM + k] = 0;
  for (int b = 0; b < DIAG_BLOCKS; ++b) {
    for (int k = 0; k < DIAG_NSUM; ++k) s[k] += part[(size_t)b * DIAG_NVAL + k];
    for (int k = 0; k < DIAG_NMAX; ++k)
      out10[DIAG_NSUM + k] = std::fmax(out10[DIAG_NSUM + k], part[(size_t)b * DIAG_NVAL + DIAG_NSUM + k]);
  }
  for (int k = 0; k < DIAG_NSUM; ++k) out10[k] = (double)s[k];
  return COSENU_OK;
}
// (4) whole-grid sums / maxima -> the diagnostics; set_reference stores the t = 0 values
void diag_finish(cosenu* h, const double* g, int set_reference, cosenu_diag_t* d) {
  const double* sums = g;
  const double* maxs = g + DIAG_NSUM;
  if (set_reference) {
    h->sum_ee0[0] = sums[0]; h->sum_ee0[1] = sums[1];
    for (int m = 0; m < 3; ++m) h->M0_init[m] = sums[3 + m] * (h->dz * h->dv);
  }
  if (!d) return;
  d->t = h->t; d->step = h->step;
  d->psurv_nu = h->sum_ee0[0] != 0 ? sums[0] / h->sum_ee0[0] : 0.0;
  d->psurv_nubar = h->sum_ee0[1] != 0 ? sums[1] / h->sum_ee0[1] : 0.0;
  d->dP_max = maxs[0];
  d->dP_avg = h->pref_sum_nu > 0 ? sums[2] / h->pref_sum_nu : 0.0;
  for (int m = 0; m < 3; ++m) { d->M0[m] = sums[3 + m] * (h->dz * h->dv); d->dM0[m] = d->M0[m] - h->M0_init[m]; }
  d->trace_dev_max = maxs[1];
  d->ex_abs_max = maxs[2];
}

// after U has been uploaded: ghosts, moments, diagnostic references
int finish_upload(cosenu* h, double t) {
  if (!h->slab) {
    fill_ghosts_kernel<<<64, 256, 0, h->stream>>>(h->U, h->nz, h->nvp, h->comp_stride, G);
    CK(cudaGetLastError());
    h->launches++;
  }
  h->mcur = 0;
  moments_kernel<<<592, 256, 0, h->stream>>>(h->U, h->M[0], h->nz, h->nv, h->nvp, h->comp_stride, G, h->dv, h->voff,
                                             h->quad);
  CK(cudaGetLastError());
  h->launches++;
  h->t = t; h->step = 0; h->have_state = true;
  if (h->slab) {   // ghost rows and references need the other slabs: slab_push_ghosts, slab_*_sums
    h->ghosts_pushed = false;
    CK(cudaStreamSynchronize(h->stream));
    return COSENU_OK;
  }
  std::vector<double> rs(4 * (size_t)h->nv);
  int rc;
  if ((rc = ref_sums(h, rs.data()))) return rc;
  if ((rc = set_ref_sums(h, rs.data()))) return rc;
  double g[DIAG_NVAL];
  if ((rc = diag_sums(h, g))) return rc;
  diag_finish(h, g, 1, nullptr);
  return COSENU_OK;
}

inline uint64_t splitmix64_next(uint64_t& s) {
  uint64_t z = (s += 0x9E3779B97F4A7C15ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

}  // namespace

namespace {
constexpr int GRAPH_STEPS = 8;

void drop_graph(cosenu* h) {
  if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
}

// capture GRAPH_STEPS steps of the current configuration into an executable graph
int build_graph(cosenu* h) {
  h->dry_run = true;                     // kernel attributes first: nothing but launches inside the capture
  for (int k = 0; k < 4; ++k) { int rc = rk_stage(h, k); if (rc) { h->dry_run = false; return rc; } }
  h->dry_run = false;
  const int64_t launches0 = h->launches, step0 = h->step;
  const double t0 = h->t;
  const unsigned long long epoch0 = h->epoch;
  CK(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
  int rc = COSENU_OK;
  for (int s = 0; s < GRAPH_STEPS && rc == COSENU_OK; ++s) rc = one_step(h);
  cudaGraph_t graph = nullptr;
  cudaError_t e = cudaStreamEndCapture(h->stream, &graph);
  h->launches = launches0; h->step = step0; h->t = t0; h->epoch = epoch0;   // nothing has run yet
  if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
  if (e != cudaSuccess) return cuda_fail(h, e, "cudaStreamEndCapture");
  e = cudaGraphInstantiate(&h->gexec, graph, 0);
  cudaGraphDestroy(graph);
  if (e != cudaSuccess) { h->gexec = nullptr; return cuda_fail(h, e, "cudaGraphInstantiate"); }
  return COSENU_OK;
}
}  // namespace

// ================================================================================ C ABI
namespace {
cosenu* create_common(int64_t nz_global, int64_t z_begin, int64_t nz, int32_t nv, double L, double dt, double omega,
                      double theta, double mu, int scheme, bool slab) {
  if (nz < 16 || nz > 2000000000ll || nz_global < nz || nz_global > 2000000000ll || z_begin < 0 || z_begin + nz > nz_global ||
      nv < 2 || nv > (1 << 20) || !(L > 0) || !(dt > 0) || (scheme != 0 && scheme != 1) || !std::isfinite(L) ||
      !std::isfinite(dt) || !std::isfinite(omega) || !std::isfinite(theta) || !std::isfinite(mu)) {
    g_create_err = "cosenu_create: invalid argument";
    return nullptr;
  }
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { g_create_err = std::string("cosenu_create: no CUDA device: ") + cudaGetErrorString(e); return nullptr; }
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, dev);
  if (e != cudaSuccess) { g_create_err = std::string("cosenu_create: ") + cudaGetErrorString(e); return nullptr; }
  if (prop.major != 10) {
    g_create_err = "cosenu_create: this library holds sm_100a code only; device is sm_" + std::to_string(prop.major) +
                   std::to_string(prop.minor);
    return nullptr;
  }
  cosenu* h = new (std::nothrow) cosenu();
  if (!h) { g_create_err = "out of memory"; return nullptr; }
  h->nz = nz; h->nv = nv; h->L = L; h->dt = dt; h->omega = omega; h->theta = theta; h->mu = mu; h->scheme = scheme;
  h->slab = slab; h->nz_global = nz_global; h->z_begin = z_begin;
  h->device = dev;
  h->nvp = (nv + 3) / 4 * 4;
  h->dz = L / (double)nz_global; h->dv = 2.0 / (double)nv;
  h->comp_stride = (int64_t)(nz + 2 * G) * h->nvp;
  h->num_sms = prop.multiProcessorCount;
  return h;
}
}  // namespace

extern "C" cosenu_t* cosenu_create(int64_t nz, int32_t nv, double L, double dt, double omega, double theta, double mu,
                                   int scheme) {
  return create_common(nz, 0, nz, nv, L, dt, omega, theta, mu, scheme, false);
}

extern "C" cosenu_t* cosenu_create_slab(int64_t nz_global, int64_t z_begin, int64_t nz_local, int32_t nv, double L,
                                        double dt, double omega, double theta, double mu, int scheme) {
  return create_common(nz_global, z_begin, nz_local, nv, L, dt, omega, theta, mu, scheme, true);
}

extern "C" size_t cosenu_workspace_bytes(const cosenu_t* h) {
  if (!h) return 0;
  size_t off[11];
  return workspace_layout(h, off);
}

extern "C" int cosenu_attach(cosenu_t* h, void* dev_workspace, size_t bytes, void* cuda_stream) {
  if (!h) return COSENU_EINVAL;
  if (h->maps_ready) return fail(h, COSENU_ESTATE, "cosenu_attach: workspace already in use");
  DeviceGuard dg_(h->device);
  if (dev_workspace) {
    if (bytes < cosenu_workspace_bytes(h) || (reinterpret_cast<uintptr_t>(dev_workspace) & 255))
      return fail(h, COSENU_EINVAL, "cosenu_attach: workspace too small or not 256-byte aligned");
    // the kernels and the TMA descriptors need plain device memory of the handle's device
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, dev_workspace);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return cuda_fail(h, e, "cosenu_attach: cudaPointerGetAttributes"); }
    if (at.type != cudaMemoryTypeDevice || at.device != h->device)
      return fail(h, COSENU_EINVAL, "cosenu_attach: the workspace is not device memory of the device the handle was created on");
    h->ws = dev_workspace; h->ws_bytes = bytes; h->ws_owned = false;
  }
  h->stream = static_cast<cudaStream_t>(cuda_stream);
  return COSENU_OK;
}

extern "C" int cosenu_set_option(cosenu_t* h, int key, double value) {
  if (!h) return COSENU_EINVAL;
  // a pure setter until the handle has touched CUDA: graph, events and tensor maps exist only after ensure_workspace
  DeviceGuard dg_(h->device, h->maps_ready || h->gexec != nullptr || !h->ev_pool.empty());
  drop_graph(h);   // the captured launch parameters may change
  switch (key) {
    case COSENU_OPT_GRAPH: h->use_graph = value != 0; return COSENU_OK;
    case COSENU_OPT_EPS_KO: if (!(value >= 0) || !std::isfinite(value)) break; h->eps_ko = value; return COSENU_OK;
    case COSENU_OPT_WENO_EPS: if (!(value >= 1e-40) || !(value <= 1e30)) break; h->weno_eps = value; return COSENU_OK;   // range of the product form, weno7_math.h
    case COSENU_OPT_MAX_CTAS: if (!(value >= 0) || !(value <= 65535) || value != std::floor(value)) break; h->max_ctas = (int)value; return COSENU_OK;
    case COSENU_OPT_HALO_TIMEOUT_S: if (!(value >= 1e-3) || !(value <= 3600.0)) break; h->halo_timeout_s = value; return COSENU_OK;
    case COSENU_OPT_ADVECT: h->advect = value != 0; return COSENU_OK;
    case COSENU_OPT_RK_FORM: if (value != 0 && value != 1 && value != 2 && value != 3) break; h->rk_form = (int)value; return COSENU_OK;
    case COSENU_OPT_VARIANT: if (value != 0 && value != 1 && value != 2 && value != 3 && value != 4) break; h->variant = (int)value; return COSENU_OK;
    case COSENU_OPT_KO_ORDER:
      if (value != 2 && value != 3) break;
      if (h->ko_r != (int)value) {
        h->ko_r = (int)value;
        if (h->maps_ready) { int rc = make_maps(h); if (rc) return rc; }   // the stage-input boxes carry the halo
      }
      return COSENU_OK;
    case COSENU_OPT_QUADRATURE:
      if ((value != 0 && value != 1 && value != 2) || (value == 2 && (h->nv % 2 == 0 || h->nv < 3))) break;
      if (h->have_state) return fail(h, COSENU_ESTATE, "cosenu_set_option: the quadrature must be chosen before init / set_state");
      h->quad = (int)value;
      h->voff = h->quad == 0 ? 0.5 : 0.0;
      h->dv = h->quad == 0 ? 2.0 / (double)h->nv : 2.0 / (double)(h->nv - 1);
      return COSENU_OK;
    case COSENU_OPT_STAGE_TIMING: {
      int rc = drain_events(h);
      if (rc) return rc;
      h->stage_timing = value != 0;
      for (int k = 0; k < 4; ++k) h->stage_ms[k] = 0;
      h->stage_n = 0;
      return COSENU_OK;
    }
  }
  return fail(h, COSENU_EINVAL, "cosenu_set_option: bad key or value");
}

extern "C" int cosenu_set_state(cosenu_t* h, const double* host_state, double t) {
  if (!h || !host_state || !std::isfinite(t)) return h ? fail(h, COSENU_EINVAL, "cosenu_set_state: invalid argument") : COSENU_EINVAL;
  DeviceGuard dg_(h->device);
  int rc = ensure_workspace(h);
  if (rc) return rc;
  for (int c = 0; c < 8; ++c) {
    CK(cudaMemcpy2DAsync(h->U + c * h->comp_stride + (size_t)G * h->nvp, sizeof(double) * h->nvp,
                         host_state + (size_t)c * h->nz * h->nv, sizeof(double) * h->nv, sizeof(double) * h->nv,
                         (size_t)h->nz, cudaMemcpyHostToDevice, h->stream));
  }
  return finish_upload(h, t);
}

extern "C" int cosenu_init(cosenu_t* h, uint64_t seed, double sigma_nu, double sigma_nubar, double alpha, double pert_amp,
                           int pert_kind) {
  if (!h) return COSENU_EINVAL;
  if (!(sigma_nu > 0) || !(sigma_nubar > 0) || !(alpha >= 0) || !std::isfinite(pert_amp) || pert_kind < 0 || pert_kind > 2)
    return fail(h, COSENU_EINVAL, "cosenu_init: invalid argument");
  const int nv = h->nv; const int64_t nz = h->nz;
  // Eq. (20), normalised so that sum_j g_j dv = 1; g_bar carries alpha
  std::vector<double> g(nv), gb(nv);
  double sg = 0, sgb = 0;
  for (int j = 0; j < nv; ++j) {
    const double v = -1.0 + ((double)j + h->voff) * h->dv, w = quad_weight(j, nv, h->quad);
    g[j] = std::exp(-(v - 1.0) * (v - 1.0) / (2.0 * sigma_nu * sigma_nu));
    gb[j] = std::exp(-(v - 1.0) * (v - 1.0) / (2.0 * sigma_nubar * sigma_nubar));
    sg += w * g[j]; sgb += w * gb[j];
  }
  for (int j = 0; j < nv; ++j) { g[j] = g[j] / (sg * h->dv); gb[j] = alpha * (gb[j] / (sgb * h->dv)); }
  const double two_pi = 6.283185307179586476925286766559;
  std::vector<double> pr(nz), pi(nz), dd(nz, 1.0);
  // a slab builds its own rows of the global initial state: global row zg = z_begin + i of nzg rows
  const int64_t z0 = h->z_begin, nzg = h->nz_global;
  uint64_t s = seed;
  if (pert_kind == 0) {
    s += (uint64_t)z0 * 0x9E3779B97F4A7C15ull;   // splitmix64's state advances by a constant per draw: skip z0 draws
    for (int64_t i = 0; i < nz; ++i) {
      const double u = (double)(splitmix64_next(s) >> 11) * (1.0 / 9007199254740992.0);
      pr[i] = pert_amp * std::cos(two_pi * u); pi[i] = pert_amp * std::sin(two_pi * u);
    }
  } else if (pert_kind == 1) {
    const int K = 16; double ph[K];
    for (int q = 0; q < K; ++q) ph[q] = two_pi * ((double)(splitmix64_next(s) >> 11) * (1.0 / 9007199254740992.0));
    for (int64_t i = 0; i < nz; ++i) {
      double a = 0, b = 0;
      for (int q = 0; q < K; ++q) {
        const double arg = two_pi * (double)(q + 1) * (double)(z0 + i) / (double)nzg + ph[q];
        a += std::cos(arg); b += std::sin(arg);
      }
      pr[i] = pert_amp * a / 4.0; pi[i] = pert_amp * b / 4.0;
    }
  } else {
    for (int64_t i = 0; i < nz; ++i) {
      const double zc = (h->scheme == COSENU_FV_WENO7 ? ((z0 + i) + 0.5) : (double)(z0 + i)) * h->dz - 0.5 * h->L;
      const double e = pert_amp * std::exp(-zc * zc / 50.0);
      pr[i] = 0.5 * e; pi[i] = 0.0; dd[i] = std::sqrt(1.0 - e * e);
    }
  }
  // The state is the outer product of these vectors: the host holds O(nz + nv) numbers and the device expands them
  // (init_expand_kernel; each entry one product, rounded once, exactly as a host loop over all cells would).
  // Scratch on the device: the 4 nz-vectors go into the moment buffer that the first stage launch overwrites, the 2
  // nv-vectors into the diagnostics partials that finish_upload overwrites.
  std::vector<double> zv(4 * (size_t)nz), gv(2 * (size_t)nv);
  for (int64_t i = 0; i < nz; ++i) {
    zv[i] = 1.0 + dd[i]; zv[(size_t)nz + i] = 1.0 - dd[i]; zv[2 * (size_t)nz + i] = pr[i]; zv[3 * (size_t)nz + i] = pi[i];
  }
  for (int j = 0; j < nv; ++j) { gv[j] = g[j]; gv[(size_t)nv + j] = gb[j]; }
  DeviceGuard dg_(h->device);
  int rc = ensure_workspace(h);
  if (rc) return rc;
  double* d_zv = h->M[1];
  double* d_gv = h->d_refpart;
  static_assert(REF_BLOCKS * 4 >= 2, "the diagnostics partials hold the two beam vectors");
  CK(cudaMemcpyAsync(d_zv, zv.data(), sizeof(double) * zv.size(), cudaMemcpyHostToDevice, h->stream));
  CK(cudaMemcpyAsync(d_gv, gv.data(), sizeof(double) * gv.size(), cudaMemcpyHostToDevice, h->stream));
  const unsigned blocks = (unsigned)(nz < 4 * (int64_t)h->num_sms * 8 ? nz : 4 * (int64_t)h->num_sms * 8);
  init_expand_kernel<<<blocks, 256, 0, h->stream>>>(h->U, d_zv, d_gv, nz, nv, h->nvp, h->comp_stride, G);
  CK(cudaGetLastError());
  h->launches++;
  rc = finish_upload(h, 0.0);     // synchronises the stream: zv / gv are no longer needed when it returns
  return rc;
}

extern "C" int cosenu_step(cosenu_t* h, int64_t n) {
  if (!h || n < 0) return h ? fail(h, COSENU_EINVAL, "cosenu_step: n < 0") : COSENU_EINVAL;
  if (!h->have_state) return fail(h, COSENU_ESTATE, "cosenu_step: no state, call cosenu_init or cosenu_set_state first");
  if (h->slab && !(h->linked && h->ghosts_pushed))
    return fail(h, COSENU_ESTATE, "cosenu_step: a slab must be linked (cosenu_slab_link) and its ghost rows exchanged "
                                  "(cosenu_slab_push_ghosts) first");
  DeviceGuard dg_(h->device);
  if (h->use_graph && !h->slab && !h->stage_timing && n >= 2 * GRAPH_STEPS) {
    if (!h->gexec && build_graph(h) != COSENU_OK) {
      // capture not possible here (e.g. a caller stream that is itself being captured): launch kernel by kernel from now on
      (void)cudaGetLastError();
      h->use_graph = 0;
    }
    for (; h->gexec && n >= GRAPH_STEPS; n -= GRAPH_STEPS) {
      CK(cudaGraphLaunch(h->gexec, h->stream));
      h->launches += 4 * GRAPH_STEPS; h->epoch += 4 * GRAPH_STEPS;
      h->step += GRAPH_STEPS;
      for (int s = 0; s < GRAPH_STEPS; ++s) h->t += h->dt;   // same rounding as step-by-step accumulation
    }
  }
  for (int64_t s = 0; s < n; ++s) {
    int rc = one_step(h);
    if (rc) return rc;
  }
  return COSENU_OK;
}

extern "C" int cosenu_sync(cosenu_t* h) {
  if (!h) return COSENU_EINVAL;
  DeviceGuard dg_(h->device);
  CK(cudaStreamSynchronize(h->stream));
  return halo_check(h, "cosenu_sync");
}

extern "C" int cosenu_get_state(cosenu_t* h, double* host_out) {
  if (!h || !host_out) return COSENU_EINVAL;
  if (!h->have_state) return fail(h, COSENU_ESTATE, "cosenu_get_state: no state");
  DeviceGuard dg_(h->device);
  for (int c = 0; c < 8; ++c) {
    CK(cudaMemcpy2DAsync(host_out + (size_t)c * h->nz * h->nv, sizeof(double) * h->nv,
                         h->U + c * h->comp_stride + (size_t)G * h->nvp, sizeof(double) * h->nvp, sizeof(double) * h->nv,
                         (size_t)h->nz, cudaMemcpyDeviceToHost, h->stream));
  }
  CK(cudaStreamSynchronize(h->stream));
  return halo_check(h, "cosenu_get_state");
}

extern "C" int cosenu_get_moments(cosenu_t* h, double* host_out) {
  if (!h || !host_out) return COSENU_EINVAL;
  if (!h->have_state) return fail(h, COSENU_ESTATE, "cosenu_get_moments: no state");
  DeviceGuard dg_(h->device);
  CK(cudaMemcpyAsync(host_out, h->M[h->mcur], sizeof(double) * 6 * (size_t)h->nz, cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return COSENU_OK;
}

extern "C" int cosenu_diagnostics(cosenu_t* h, cosenu_diag_t* d) {
  if (!h || !d) return COSENU_EINVAL;
  if (!h->have_state) return fail(h, COSENU_ESTATE, "cosenu_diagnostics: no state");
  if (h->slab) return fail(h, COSENU_ESTATE, "cosenu_diagnostics: a slab holds part of the grid; use cosenu_slab_diag_sums + "
                                             "a reduction over the slabs + cosenu_slab_diag_finish");
  DeviceGuard dg_(h->device);
  double g[DIAG_NVAL];
  int rc = diag_sums(h, g);
  if (rc) return rc;
  diag_finish(h, g, 0, d);
  return COSENU_OK;
}

extern "C" int64_t cosenu_launch_count(const cosenu_t* h) { return h ? h->launches : 0; }

extern "C" int cosenu_stage_times(cosenu_t* h, double* ms_sum, int64_t* launches_per_stage) {
  if (!h || !ms_sum || !launches_per_stage) return COSENU_EINVAL;
  DeviceGuard dg_(h->device);
  int rc = drain_events(h);
  if (rc) return rc;
  for (int k = 0; k < 4; ++k) { ms_sum[k] = h->stage_ms[k]; h->stage_ms[k] = 0; }
  *launches_per_stage = h->stage_n; h->stage_n = 0;
  return COSENU_OK;
}

extern "C" void cosenu_destroy(cosenu_t* h) {
  if (!h) return;
  DeviceGuard dg_(h->device);
  if (h->maps_ready) cudaStreamSynchronize(h->stream);
  for (cudaEvent_t e : h->ev_pool) cudaEventDestroy(e);
  drop_graph(h);
  for (int k = 0; k < 2; ++k)
    if (h->ipc_mapped[k] && (k == 0 || h->ipc_mapped[1] != h->ipc_mapped[0])) cudaIpcCloseMemHandle(h->ipc_mapped[k]);
  if (h->ws_owned && h->ws) cudaFree(h->ws);
  if (h->stream_owned) cudaStreamDestroy(h->stream);
  delete h;
}

extern "C" const char* cosenu_last_error(const cosenu_t* h) { return h ? h->err.c_str() : g_create_err.c_str(); }

#ifndef COSENU_BUILD_ID
#define COSENU_BUILD_ID "unknown"   // built by hand, without paper_2203_12866_b200/build.py
#endif
extern "C" const char* cosenu_build_id(void) { return COSENU_BUILD_ID; }

// ================================================================================ z-slab decomposition
namespace {
typedef CUresult (*PFN_getAddressRange)(CUdeviceptr*, size_t*, CUdeviceptr);
}

extern "C" int cosenu_slab_export(cosenu_t* h, cosenu_slab_peer_t* out) {
  if (!h || !out) return COSENU_EINVAL;
  if (!h->slab) return fail(h, COSENU_ESTATE, "cosenu_slab_export: not a slab handle (cosenu_create_slab)");
  DeviceGuard dg_(h->device);
  int rc = ensure_workspace(h);
  if (rc) return rc;
  CK(cudaStreamSynchronize(h->stream));   // the workspace is zeroed (counters start at 0) before anybody can reach it
  std::memset(out, 0, sizeof(*out));
  // the IPC handle names the whole allocation: find its base (a caller-owned workspace may sit inside a larger one)
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qr;
  CK(cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &qr));
  CUdeviceptr base = 0; size_t size = 0;
  if (!fn || qr != cudaDriverEntryPointSuccess ||
      reinterpret_cast<PFN_getAddressRange>(fn)(&base, &size, (CUdeviceptr)h->ws) != CUDA_SUCCESS)
    return fail(h, COSENU_ECUDA, "cosenu_slab_export: cuMemGetAddressRange failed");
  cudaIpcMemHandle_t ipc;
  cudaError_t e = cudaIpcGetMemHandle(&ipc, (void*)base);
  if (e == cudaSuccess) {
    static_assert(sizeof(ipc) == 64, "cudaIpcMemHandle_t");
    std::memcpy(out->ipc_handle, &ipc, 64);
  } else {
    (void)cudaGetLastError();   // not shareable (e.g. a pooled allocation): the slab can still be linked inside this process
  }
  out->ipc_offset = (uint64_t)((CUdeviceptr)h->ws - base);
  out->dev_base = (uint64_t)(uintptr_t)h->ws;
  out->pid = (int64_t)getpid();
  out->device = h->device;
  out->nvp = h->nvp;
  out->nz_local = h->nz;
  out->comp_stride = h->comp_stride;
  const char* b = static_cast<const char*>(h->ws);
  out->off_buf[0] = (uint64_t)((const char*)h->U - b); out->off_buf[1] = (uint64_t)((const char*)h->Y1 - b);
  out->off_buf[2] = (uint64_t)((const char*)h->Y2 - b); out->off_buf[3] = (uint64_t)((const char*)h->ACC - b);
  out->off_ctr = (uint64_t)((const char*)h->d_ctr - b);
  return COSENU_OK;
}

extern "C" int cosenu_slab_link(cosenu_t* h, const cosenu_slab_peer_t* lo, const cosenu_slab_peer_t* hi) {
  if (!h || !lo || !hi) return COSENU_EINVAL;
  if (!h->slab) return fail(h, COSENU_ESTATE, "cosenu_slab_link: not a slab handle");
  if (h->linked) return fail(h, COSENU_ESTATE, "cosenu_slab_link: already linked");
  DeviceGuard dg_(h->device);   // peer access is enabled FROM the current device, IPC handles are opened on it
  int rc = ensure_workspace(h);
  if (rc) return rc;
  const cosenu_slab_peer_t* peers[2] = {lo, hi};
  for (int k = 0; k < 2; ++k) {
    const cosenu_slab_peer_t* q = peers[k];
    if (q->nvp != h->nvp || q->nz_local < 16) return fail(h, COSENU_EINVAL, "cosenu_slab_link: neighbour has another v-grid or is too thin");
    char* base = nullptr;
    if (q->pid == (int64_t)getpid()) {
      base = reinterpret_cast<char*>((uintptr_t)q->dev_base);
      if (q->device != h->device) {   // another GPU of this process: direct peer access
        cudaError_t e = cudaDeviceEnablePeerAccess(q->device, 0);
        if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) return cuda_fail(h, e, "cudaDeviceEnablePeerAccess");
        (void)cudaGetLastError();
      }
    } else if (k == 1 && lo->pid == hi->pid && std::memcmp(lo->ipc_handle, hi->ipc_handle, 64) == 0 && h->ipc_mapped[0]) {
      h->ipc_mapped[1] = h->ipc_mapped[0];   // two slabs in a ring: both neighbours are the same allocation
      base = static_cast<char*>(h->ipc_mapped[1]) + q->ipc_offset;
    } else {
      cudaIpcMemHandle_t ipc;
      std::memcpy(&ipc, q->ipc_handle, 64);
      void* mapped = nullptr;
      cudaError_t e = cudaIpcOpenMemHandle(&mapped, ipc, cudaIpcMemLazyEnablePeerAccess);
      if (e != cudaSuccess) return cuda_fail(h, e, "cudaIpcOpenMemHandle (neighbouring slab)");
      h->ipc_mapped[k] = mapped;
      base = static_cast<char*>(mapped) + q->ipc_offset;
    }
    for (int b = 0; b < 4; ++b) h->peer_buf[k][b] = reinterpret_cast<double*>(base + q->off_buf[b]);
    h->peer_stride[k] = q->comp_stride;
    h->peer_nz[k] = q->nz_local;
    // my low rows land in the lower slab's HIGH ghost rows (its counter [1]); my high rows in the upper slab's LOW ones ([0])
    h->peer_ctr[k] = reinterpret_cast<unsigned long long*>(base + q->off_ctr) + (k == 0 ? 1 : 0);
  }
  h->linked = true;
  h->epoch = 0;
  return COSENU_OK;
}

extern "C" int cosenu_slab_push_ghosts(cosenu_t* h) {
  if (!h) return COSENU_EINVAL;
  if (!h->slab || !h->linked) return fail(h, COSENU_ESTATE, "cosenu_slab_push_ghosts: slab not linked");
  if (!h->have_state) return fail(h, COSENU_ESTATE, "cosenu_slab_push_ghosts: no state");
  DeviceGuard dg_(h->device);
  push_ghosts_kernel<<<64, 256, 0, h->stream>>>(h->U, h->nz, h->nvp, h->comp_stride, G,
                                                h->peer_buf[0][0] + (size_t)(h->peer_nz[0] + G) * h->nvp, h->peer_stride[0],
                                                h->peer_buf[1][0], h->peer_stride[1]);
  CK(cudaGetLastError());
  h->launches++;
  CK(cudaStreamSynchronize(h->stream));
  h->ghosts_pushed = true;
  return COSENU_OK;
}

extern "C" int cosenu_slab_ref_sums(cosenu_t* h, double* out) {
  if (!h || !out) return COSENU_EINVAL;
  if (!h->have_state) return fail(h, COSENU_ESTATE, "cosenu_slab_ref_sums: no state");
  DeviceGuard dg_(h->device);
  return ref_sums(h, out);
}

extern "C" int cosenu_slab_set_ref_sums(cosenu_t* h, const double* global_sums) {
  if (!h || !global_sums) return COSENU_EINVAL;
  if (!h->have_state) return fail(h, COSENU_ESTATE, "cosenu_slab_set_ref_sums: no state");
  DeviceGuard dg_(h->device);
  return set_ref_sums(h, global_sums);
}

extern "C" int cosenu_slab_diag_sums(cosenu_t* h, double* out10) {
  if (!h || !out10) return COSENU_EINVAL;
  if (!h->have_state) return fail(h, COSENU_ESTATE, "cosenu_slab_diag_sums: no state");
  DeviceGuard dg_(h->device);
  int rc = diag_sums(h, out10);
  return rc ? rc : halo_check(h, "cosenu_slab_diag_sums");
}

extern "C" int cosenu_slab_diag_finish(cosenu_t* h, const double* global10, int set_reference, cosenu_diag_t* out) {
  if (!h || !global10) return COSENU_EINVAL;
  if (!h->have_state) return fail(h, COSENU_ESTATE, "cosenu_slab_diag_finish: no state");
  diag_finish(h, global10, set_reference, out);
  return COSENU_OK;
}

extern "C" int cosenu_slab_step_group(cosenu_t** hs, int32_t count, int64_t n) {
  if (!hs || count < 1 || n < 0) return COSENU_EINVAL;
  for (int i = 0; i < count; ++i) {
    cosenu* h = hs[i];
    if (!h) return COSENU_EINVAL;
    if (!h->slab || !h->linked || !h->ghosts_pushed || !h->have_state)
      return fail(h, COSENU_ESTATE, "cosenu_slab_step_group: every slab must be linked, hold a state and have its ghosts exchanged");
    if (h->stream != hs[0]->stream || h->device != hs[0]->device)
      return fail(h, COSENU_EINVAL, "cosenu_slab_step_group: the slabs of a group share one device and one stream");
  }
  DeviceGuard dg_(hs[0]->device);
  for (int64_t s = 0; s < n; ++s) {
    for (int k = 0; k < 4; ++k)
      for (int i = 0; i < count; ++i) {
        int rc = rk_stage(hs[i], k);
        if (rc) return rc;
      }
    for (int i = 0; i < count; ++i) { hs[i]->t += hs[i]->dt; hs[i]->step += 1; }
  }
  return COSENU_OK;
}

extern "C" int cosenu_slab_stage(cosenu_t* h, int32_t k) {
  if (!h || k < 0 || k > 3) return h ? fail(h, COSENU_EINVAL, "cosenu_slab_stage: k must be 0..3") : COSENU_EINVAL;
  if (!h->slab || !h->linked || !h->ghosts_pushed || !h->have_state)
    return fail(h, COSENU_ESTATE, "cosenu_slab_stage: the slab must be linked, hold a state and have its ghosts exchanged");
  DeviceGuard dg_(h->device);
  int rc = rk_stage(h, k);
  if (rc) return rc;
  if (k == 3) { h->t += h->dt; h->step += 1; }
  return COSENU_OK;
}

extern "C" int cosenu_slab_wait_failed(cosenu_t* h, int32_t* failed) {
  if (!h || !failed) return COSENU_EINVAL;
  if (!h->maps_ready) { *failed = 0; return COSENU_OK; }
  DeviceGuard dg_(h->device);
  int v = 0;
  CK(cudaMemcpyAsync(&v, h->d_err, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  *failed = v;
  return COSENU_OK;
}
