// stage_kernels.cuh -- ONE fused, persistent kernel per RK stage (sm_100a, fp64).
//
// Per launch and per (z,v) cell:
//   advection of the 8 real components by FD4+KO3 or FV-WENO7 (App. A),
//   Hamiltonian from the 6 per-z velocity moments of the stage input (Eq. 3a/3b),
//   commutator -i[H,rho], -i[Hbar,rhobar] (Eq. 1a/1b),
//   classical RK4 combine,
//   and, in the epilogue, the 6 velocity moments of the state just produced (the S1 of the next stage).
//
// Design.  Device layout of a state: double [8][nz + 2G][nvp], v fastest (G = 4
// periodic ghost rows on each side of z, nvp = nv rounded up to 4).
//  * Persistent CTAs (one per SM).  Work item = (z-tile of TZ rows, chunk of 32 beams); a CTA walks the
//    chunks of its tiles (tile = blockIdx.x + k gridDim.x), so a tile's moments never leave the CTA.
//  * Warp-specialised: one producer warp feeds shared memory with 3-D TMA boxes (cp.async.bulk.tensor):
//    the stage-input tile with its stencil halo [8][TZ+2H][32] (ring of NY slots) and the operands that
//    have no reuse, u0 and the RK accumulator [8][TZ][32] (ring of NUA slots); full/empty mbarriers.
//    The compute warps never wait on a global load.
//  * Compute warp w owns rows w*S .. w*S+S-1 of the tile, lane = beam.  WENO7: every interface flux is
//    computed once; neighbouring warps exchange the flux of their common interface through shared memory
//    (xfull/xfree mbarriers); the tile's left boundary flux is split by component over 8 warps.
//  * Moments of the output: butterfly reduce-scatter over the lanes (N values cost ~N adds, not 5N),
//    accumulated over the chunks in registers of the owning lanes in fixed order => bit-reproducible.
//  * Tile heights and warps: TZ = 16 with 8 compute warps x 2 rows everywhere, except the WENO7 kernels of the default RK
//    form, which run three compute warps per scheduler as far as shared memory and registers allow: 12 warps x 2 rows
//    (TZ = 24), 11 x 2 (TZ = 22) or, with two staged arrays, 10 x 2 (TZ = 20).  SCHEME 2 = FD4 + KO of order r = 3 (halo 3).
//  * Ghost rows / z-slabs: the warps that produce the first / last G rows also store their ghost copies -- into this
//    buffer (periodic domain) or into the neighbouring slab's buffer over peer memory, followed by a release-add on
//    the neighbour's arrival counter; the DMA warp acquires its own counters before it loads a tile that touches ghost
//    rows.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "aux_kernels.cuh"
#include "weno7_math.h"

namespace cosenu_dev {

constexpr int G = 4;    // ghost rows per side in the device layout
constexpr int VC = 32;  // beams per chunk = lanes of a warp

// RK4 formulations:
//  accumulator form  : FIRST, MID, MID, LAST                    1024 B per cell-step
//  lean accumulator  : FIRST_LEAN, MID_REBUILD, MID, LAST        896 B
//  accumulator-free  : FIRST_LEAN, MID_NOACC, MID_NOACC, LAST_COMB   832 B:
//      Y2 = U + dt/2 k1, Y3 = U + dt/2 k2, Y4 = U + dt k3,  U+ = (Y2 + 2 Y3 + Y4 - U)/3 + dt/6 k4
//  partial sum       : FIRST_LEAN, MID_P, MID_NOACC, LAST_P            768 B:
//      stage 2 also stores P = (Y2 + 2 Y3 - U)/3 (it holds all three); stage 4 reads only P: U+ = P + Y4/3 + dt/6 k4
enum StageKind { FIRST = 0, FIRST_LEAN = 1, MID = 2, MID_REBUILD = 3, LAST = 4, MID_NOACC = 5, LAST_COMB = 6, MID_P = 7,
                 LAST_P = 8 };

struct StageParams {
  double* y_out;          // next stage input (FIRST/MID) or the new U (LAST)
  double* acc_out;        // RK accumulator (FIRST, MID kinds)
  const double* mom_in;   // [6][nz] moments of the stage input (already times dv)
  double* mom_out;        // [6][nz] moments of y_out
  long long nz;
  int nv, nvp;
  long long comp_stride;  // (nz + 2G) * nvp
  double cy, ca;          // y_out = base + cy k ; acc_out = acc_in + ca k
  double mu, A0, Br0;     // A0 = -omega cos 2theta, Br0 = (omega/2) sin 2theta
  double dv, voff;         // v_j = -1 + (j + voff) dv: voff = 1/2 bin centres, 0 vertex-centred
  int quad;                // rule of the v' integral: 0 Riemann/midpoint, 1 trapezoid, 2 Simpson (aux_kernels.cuh: quad_weight)
  double cadv, cko;          // FD: -1/(12 dz), -eps_ko/(16 dz) [KO r = 2] or +eps_ko/(64 dz) [r = 3]  (times the advect switch)
  double ninv_dz, weno_eps;  // WENO: -1/dz (times the advect switch), epsilon of Eq. (14)
  // ---- ghost rows of y_out.  The copies of my first / last G rows go to
  //   ghost_lo_dst[c * ghost_lo_stride + iz * nvp + j]              (iz = 0..G-1)
  //   ghost_hi_dst[c * ghost_hi_stride + (iz - (nz - G)) * nvp + j] (iz = nz-G..nz-1)
  // single periodic domain: my own ghost rows; z-slab: the neighbouring slabs' ghost rows (peer memory).
  double* ghost_lo_dst;
  double* ghost_hi_dst;
  long long ghost_lo_stride, ghost_hi_stride;
  // z-slab only (null otherwise): arrival counters, in rows.  sig_*: the neighbours' counters, bumped (release, system
  // scope) once the ghost rows written above are visible; wait_*: my own counters, which must have reached wait_val
  // before a tile that touches the low / high ghost rows of the stage input is loaded.
  unsigned long long* sig_lo;
  unsigned long long* sig_hi;
  const unsigned long long* wait_lo;
  const unsigned long long* wait_hi;
  unsigned long long wait_val;
  int* err_flag;           // set to 1 when a wait gives up (a neighbour that never arrives must not hang the GPU)
  unsigned long long wait_timeout_ns;   // how long a halo wait may last before it gives up (COSENU_OPT_HALO_TIMEOUT_S)
  long long tile_shift;    // the l-th tile a CTA grid walks is tile (l + tile_shift) mod ntiles (slab: edge tiles first)
};

// ----------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, 0x989680;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
// 3-D tiled TMA load global -> shared, completion on an mbarrier
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
      "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
// 3-D tiled TMA store shared -> global (bulk async-group completion); out-of-range elements are clipped
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, uint32_t src, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(map), "r"(src),
               "r"(c0), "r"(c1), "r"(c2)
               : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// make this thread's shared-memory writes visible to the async proxy (TMA) before signalling
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ double lds(uint32_t addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts(uint32_t addr, double v) {
  asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}

// ---- cross-GPU arrival counters (z-slab halo exchange)
__device__ __forceinline__ unsigned long long ld_acquire_sys(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_add_release_sys(unsigned long long* p, unsigned long long v) {
  asm volatile("red.release.sys.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long global_timer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
// wait until *ctr >= val; gives up after timeout_ns (default 4 s; sets *err) so that a missing neighbour is an error, not a hang
__device__ __noinline__ void wait_arrivals(const unsigned long long* ctr, unsigned long long val, int* err,
                                           unsigned long long timeout_ns) {
  if (ld_acquire_sys(ctr) >= val) return;
  if (err && *reinterpret_cast<volatile int*>(err)) return;   // an earlier wait has already given up: the run is invalid, do not add the time-out per tile
  const unsigned long long t0 = global_timer_ns();
  while (ld_acquire_sys(ctr) < val) {
    __nanosleep(200);
    if (global_timer_ns() - t0 > timeout_ns) {
      if (err) atomicExch(err, 1);
      return;
    }
  }
}

template <int KIND>
struct KindTraits {
  static constexpr bool LOAD_U0 = (KIND == MID || KIND == MID_REBUILD || KIND == MID_NOACC || KIND == LAST_COMB || KIND == MID_P);
  static constexpr bool LOAD_ACC = (KIND == MID || KIND == LAST || KIND == LAST_P);
  static constexpr bool LOAD_Y23 = (KIND == LAST_COMB);   // the two earlier stage states Y2, Y3
  static constexpr bool WRITE_ACC = (KIND == FIRST || KIND == MID || KIND == MID_REBUILD || KIND == MID_P);
  static constexpr int NLOAD = (LOAD_U0 ? 1 : 0) + (LOAD_ACC ? 1 : 0) + (LOAD_Y23 ? 2 : 0);
  // staging arrays of one slot: array 0 = u0 on load (acc for LAST), y_out on store;
  //                             array 1 = acc on load (MID) / Y2 (LAST_COMB), acc_out on store; array 2 = Y3
  static constexpr int NARR = LOAD_Y23 ? 3 : (WRITE_ACC ? 2 : 1);
  static constexpr int ACC_LOAD_ARR = LOAD_U0 ? 1 : 0;
};

// shared-memory carve-up (byte offsets from a 128-byte aligned base)
template <int SCHEME, int KIND, int TZ, int NSEG, int NY, int NUA>
struct StageSmem {
  static constexpr int H = SCHEME == 0 ? 2 : (SCHEME == 1 ? 4 : 3);   // SCHEME 2 = FD4 + KO of order r = 3
  static constexpr int ROWS = TZ + 2 * H;
  static constexpr uint32_t YTILE = 8u * ROWS * VC * 8u;   // bytes per stage-input slot
  static constexpr uint32_t PTILE = 8u * TZ * VC * 8u;     // bytes per staging array
  static constexpr int NARR = KindTraits<KIND>::NARR;
  static constexpr uint32_t off_y = 0;
  static constexpr uint32_t off_ua = off_y + NY * YTILE;               // [NUA][NARR][PTILE]
  // copies of the flux exchange buffers (two when shared memory allows: lets neighbouring warps drift by one item)
  static constexpr int XBUF = (NSEG <= 8 && NARR < 3) ? 2 : 1;
  static constexpr uint32_t XSZ = NSEG * 8u * VC * 8u, XBSZ = 8u * VC * 8u;
  static constexpr uint32_t off_x = off_ua + NUA * NARR * PTILE;       // [XBUF][NSEG][8][32] exchange (WENO)
  static constexpr uint32_t off_xb = off_x + (SCHEME == 1 ? XBUF * XSZ : 0u);  // [XBUF][8][32] boundary (WENO)
  static constexpr uint32_t off_bar = off_xb + (SCHEME == 1 ? XBUF * XBSZ : 0u);
  // full_y[NY] empty_y[NY] full_ua[NUA] out_ready[NUA] | xf[XBUF][NSEG] xr[XBUF][NSEG] xbf[XBUF] xbr[XBUF]
  static constexpr uint32_t nbar = 2 * NY + 2 * NUA + XBUF * (2 * NSEG + 2);
  static constexpr size_t bytes = off_bar + 8 * nbar + 128;
};

// ----------------------------------------------------------------------------- butterfly reduce-scatter
// Sum each of x[0..N-1] over the 32 lanes.  Stage with lane offset o halves the live values: the lanes with
// bit o keep the upper half and send the lower half (and vice versa), so N values cost about N adds and
// N shuffles per lane instead of 5N.  On return x[0] of lane L holds the total of the original value
// `idx` (if `valid`), idx = sum over stages of (lane bit ? half : 0).  Fixed tree => reproducible.
// one stage (lane offset O, N live values -> (N + 1) / 2) and the stages below it; every index is a compile-time constant,
// so the values stay in registers whatever N is
template <int N, int O>
__device__ __forceinline__ void butterfly_stage(double* x, int lane) {
  constexpr int half = (N + 1) / 2;
  const bool up = (lane & O) != 0;
#pragma unroll
  for (int i = 0; i < half; ++i) {
    const double a = x[i];
    const double b = (i + half < N) ? x[i + half] : 0.0;
    const double send = up ? a : b;
    const double keep = up ? b : a;
    x[i] = keep + __shfl_xor_sync(0xffffffffu, send, O);
  }
  if constexpr (O > 1) butterfly_stage<half, O / 2>(x, lane);
}
template <int N>
__device__ __forceinline__ void butterfly_reduce(double (&x)[N], int lane, int& idx, bool& valid) {
  butterfly_stage<N, 16>(x, lane);
  // which original index ended up in x[0] of this lane (replay the stages backwards)
  int ns[5], hs[5];
  int n = N;
#pragma unroll
  for (int k = 0; k < 5; ++k) { ns[k] = n; hs[k] = (n + 1) / 2; n = hs[k]; }
  int pos = 0;
  valid = true;
#pragma unroll
  for (int k = 4; k >= 0; --k) {
    if (lane & (16 >> k)) pos += hs[k];
    valid = valid && (pos < ns[k]);
  }
  idx = pos;
}

// ----------------------------------------------------------------------------- WENO7 fluxes of a warp's rows
// Tw = shared address of (component 0, tile row 0 [halo included], this lane) of the stage-input tile plus
// rel_row*256: every load below then has an immediate offset.  DIR = +1 for v >= 0 (stencil biased to
// smaller z), -1 for v < 0 (mirror image about the interface, reading A9).
// FR[s][c] = WENO7 value of u_c at the right interface of row (rel_row + s).
template <int DIR, int S, int ROWS, int H>
__device__ __forceinline__ void weno_rows(uint32_t Tw, const cosenu_math::Weno7Beam& bm, double (&FR)[S][8]) {
  static_assert(S == 1 || S == 2, "rows per warp");
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    if constexpr (S == 1) {
      double w[7];
#pragma unroll
      for (int k = 0; k < 7; ++k) w[k] = lds(Tw + ((c * ROWS + H + (DIR > 0 ? 0 : 1) + DIR * (k - 3)) * VC) * 8);
      FR[0][c] = cosenu_math::weno7_face(w, bm);
    } else {
      double w[8], Fa, Fb;
#pragma unroll
      for (int k = 0; k < 8; ++k) w[k] = lds(Tw + ((c * ROWS + H + (DIR > 0 ? k - 3 : 5 - k)) * VC) * 8);
      cosenu_math::weno7_face2(w, bm, Fa, Fb);
      FR[DIR > 0 ? 0 : 1][c] = Fa;
      FR[DIR > 0 ? 1 : 0][c] = Fb;
    }
  }
}
// value at the left boundary interface of the tile (between tile rows H-1 and H) of one component
template <int DIR, int ROWS, int H>
__device__ __forceinline__ double weno_boundary(uint32_t Tc /* component base + lane */, const cosenu_math::Weno7Beam& bm) {
  double w[7];
#pragma unroll
  for (int k = 0; k < 7; ++k) w[k] = lds(Tc + ((H - 1 + (DIR > 0 ? 0 : 1) + DIR * (k - 3)) * VC) * 8);
  return cosenu_math::weno7_face(w, bm);
}
// out-of-line copies for warps whose lanes move in both directions (only the chunk that contains v = 0)
template <int DIR, int S, int ROWS, int H>
__device__ __noinline__ void weno_rows_slow(uint32_t Tw, const cosenu_math::Weno7Beam& bm, double* FRflat) {
  double FR[S][8];
  weno_rows<DIR, S, ROWS, H>(Tw, bm, FR);
#pragma unroll
  for (int s = 0; s < S; ++s)
#pragma unroll
    for (int c = 0; c < 8; ++c) FRflat[s * 8 + c] = FR[s][c];
}
template <int DIR, int ROWS, int H>
__device__ __noinline__ double weno_boundary_slow(uint32_t Tc, const cosenu_math::Weno7Beam& bm) {
  return weno_boundary<DIR, ROWS, H>(Tc, bm);
}

// ----------------------------------------------------------------------------- the stage kernel
template <int SCHEME, int KIND, int TZ, int NSEG, int NY, int NUA>
__global__ void __launch_bounds__(NSEG * 32 + 32, 1)
    stage_kernel(const __grid_constant__ CUtensorMap tm_y,     // stage input with halo: box [8][TZ+2H][32]
                 const __grid_constant__ CUtensorMap tm_u0,    // U, rows 0..nz-1: box [8][TZ][32]
                 const __grid_constant__ CUtensorMap tm_acc,   // RK accumulator (loaded and stored) / Y2 for LAST_COMB
                 const __grid_constant__ CUtensorMap tm_y3,    // Y3 for LAST_COMB
                 const __grid_constant__ CUtensorMap tm_out,   // y_out, rows 0..nz-1
                 const StageParams p) {
  using SM = StageSmem<SCHEME, KIND, TZ, NSEG, NY, NUA>;
  using KT = KindTraits<KIND>;
  constexpr int H = SM::H, ROWS = SM::ROWS;
  constexpr int S = TZ / NSEG;
  constexpr int NW = NSEG;  // compute warps
  constexpr int NARR = KT::NARR;
  static_assert(TZ % NSEG == 0 && 6 * S <= 32, "tile shape");
  static_assert(SCHEME != 1 || NSEG >= 8, "WENO boundary flux is split over 8 warps");

  extern __shared__ unsigned char smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 127u) & ~127u;
  const uint32_t s_y = sbase + SM::off_y, s_ua = sbase + SM::off_ua, s_x = sbase + SM::off_x, s_xb = sbase + SM::off_xb;
  const uint32_t s_bar = sbase + SM::off_bar;
  constexpr int XBUF = SM::XBUF;
  // barriers: full_y[NY], empty_y[NY], full_ua[NUA], out_ready[NUA]; flux exchange between neighbouring
  // warps is pairwise: xf[b][w] "warp w published its last flux", xr[b][w] "warp w+1 has read it",
  // xbf[b] "the 8 boundary pieces are published", xbr[b] "warp 0 has read them"
  const uint32_t b_full_y = s_bar, b_empty_y = s_bar + 8 * NY, b_full_ua = s_bar + 16 * NY,
                 b_out_ready = s_bar + 16 * NY + 8 * NUA, b_xf = s_bar + 16 * NY + 16 * NUA,
                 b_xr = b_xf + 8 * XBUF * NSEG, b_xbf = b_xr + 8 * XBUF * NSEG, b_xbr = b_xbf + 8 * XBUF;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nchunks = (p.nv + VC - 1) / VC;
  const long long ntiles = (p.nz + TZ - 1) / TZ;
  const long long my_tiles = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const long long nitems = my_tiles * nchunks;
  // the l-th tile of the walk (l = blockIdx.x + k gridDim.x < ntiles)
  auto tile_of = [&](long long l) { const long long t = l + p.tile_shift; return t >= ntiles ? t - ntiles : t; };

  if (threadIdx.x == 0) {
    for (int b = 0; b < NY; ++b) { mbar_init(b_full_y + 8 * b, 1); mbar_init(b_empty_y + 8 * b, NW); }
    for (int b = 0; b < NUA; ++b) { mbar_init(b_full_ua + 8 * b, 1); mbar_init(b_out_ready + 8 * b, NW); }
    if constexpr (SCHEME == 1) {
      for (int b = 0; b < XBUF * NSEG; ++b) { mbar_init(b_xf + 8 * b, 1); mbar_init(b_xr + 8 * b, 1); }
      for (int b = 0; b < XBUF; ++b) { mbar_init(b_xbf + 8 * b, 8); mbar_init(b_xbr + 8 * b, 1); }
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // =========================================================================== DMA warp (one lane)
  // item n: (1) stage-input tile into y slot n % NY once its previous readers are done;
  //         (2) outputs of item n - NUA (staged in place in slot n % NUA by the compute warps) -> global;
  //         (3) u0 / acc of item n into that slot (or just "slot is free" when the stage loads neither).
  if (warp == NW) {
    if (lane == 0) {
      auto load_stream = [&](uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1) {   // operands without reuse
        tma_load_3d(dst, map, bar, c0, c1, 0);
      };
      auto store_item = [&](long long m) {   // outputs of item m
        const int su = (int)(m % NUA);
        const int iz0 = (int)(tile_of(blockIdx.x + (m / nchunks) * gridDim.x) * TZ), c0 = (int)(m % nchunks) * VC;
        mbar_wait(b_out_ready + 8 * su, (uint32_t)((m / NUA) & 1));
        const uint32_t src = s_ua + su * NARR * SM::PTILE;
        tma_store_3d(&tm_out, src, c0, iz0, 0);
        if constexpr (KT::WRITE_ACC) tma_store_3d(&tm_acc, src + SM::PTILE, c0, iz0, 0);
        tma_store_commit();
        tma_store_wait_read();   // the slot may be overwritten from here on
      };
      long long ltile = blockIdx.x;
      int ch = 0;
      for (long long n = 0; n < nitems; ++n) {
        const long long tile = tile_of(ltile);
        const int iz0 = (int)(tile * TZ);
        const int sy = (int)(n % NY);
        if (ch == 0 && (p.wait_lo != nullptr || p.wait_hi != nullptr)) {
          // z-slab: the ghost rows this tile reads (and the neighbour's ghost rows its edge rows overwrite) belong to
          // the exchange with the neighbouring GPUs: wait for their rows of the previous stage
          bool waited = false;
          if (p.wait_lo != nullptr && tile * TZ < G) { wait_arrivals(p.wait_lo, p.wait_val, p.err_flag, p.wait_timeout_ns); waited = true; }
          if (p.wait_hi != nullptr && (tile + 1) * TZ + G > p.nz) { wait_arrivals(p.wait_hi, p.wait_val, p.err_flag, p.wait_timeout_ns); waited = true; }
          if (waited) asm volatile("fence.proxy.async.global;" ::: "memory");   // generic-proxy acquire -> TMA (async proxy) reads
        }
        mbar_wait(b_empty_y + 8 * sy, (uint32_t)(((n / NY) & 1) ^ 1));
        mbar_expect_tx(b_full_y + 8 * sy, SM::YTILE);
        tma_load_3d(s_y + sy * SM::YTILE, &tm_y, b_full_y + 8 * sy, ch * VC, iz0 + G - H, 0);
        if (n >= NUA) store_item(n - NUA);
        const int su = (int)(n % NUA);
        if constexpr (KT::NLOAD > 0) {
          mbar_expect_tx(b_full_ua + 8 * su, KT::NLOAD * SM::PTILE);
          const uint32_t dst = s_ua + su * NARR * SM::PTILE;
          if constexpr (KT::LOAD_U0) load_stream(dst, &tm_u0, b_full_ua + 8 * su, ch * VC, iz0);
          if constexpr (KT::LOAD_ACC) load_stream(dst + KT::ACC_LOAD_ARR * SM::PTILE, &tm_acc, b_full_ua + 8 * su, ch * VC, iz0);
          if constexpr (KT::LOAD_Y23) {
            load_stream(dst + SM::PTILE, &tm_acc, b_full_ua + 8 * su, ch * VC, iz0);
            load_stream(dst + 2 * SM::PTILE, &tm_y3, b_full_ua + 8 * su, ch * VC, iz0);
          }
        } else {
          mbar_arrive(b_full_ua + 8 * su);   // nothing to load: the slot is free for staging
        }
        if (++ch == nchunks) { ch = 0; ltile += gridDim.x; }
      }
      for (long long m = nitems > NUA ? nitems - NUA : 0; m < nitems; ++m) store_item(m);
      tma_store_wait_all();
    }
    return;
  }

  // =========================================================================== compute warps
  const int row0 = warp * S;
  double msum[6 * S];     // per-lane partial moments of the tile's output, summed over the chunks in order
#pragma unroll
  for (int q = 0; q < 6 * S; ++q) msum[q] = 0.0;
  // lane l < 6S holds moment (l % 6) of row row0 + l / 6 of the stage input; the next tile's values are
  // fetched one tile ahead (and only touched at the next tile) so that their latency is never exposed
  auto load_min = [&](long long l) {   // l = position in the walk
    double m = 0.0;
    if (lane < 6 * S && l < ntiles) {
      const long long iz = tile_of(l) * TZ + row0 + lane / 6;
      if (iz < p.nz) m = __ldg(p.mom_in + (long long)(lane % 6) * p.nz + iz);
    }
    return m;
  };
  double min_cur = 0.0, min_next = load_min(blockIdx.x);
  long long ltile = blockIdx.x;
  int ch = 0;
  for (long long n = 0; n < nitems; ++n) {
    const long long iz0 = tile_of(ltile) * TZ;
    if (ch == 0) {
      min_cur = p.mu * min_next;
      min_next = load_min(ltile + gridDim.x);
    }
    const int sy = (int)(n % NY), su = (int)(n % NUA);
    const uint32_t Ty = s_y + sy * SM::YTILE + lane * 8;                  // + ((c * ROWS + r) * 32) * 8
    const uint32_t Tu = s_ua + su * NARR * SM::PTILE + lane * 8;          // + ((c * TZ + r) * 32) * 8
    const uint32_t Ta_in = Tu + KT::ACC_LOAD_ARR * SM::PTILE, Ta_out = Tu + SM::PTILE;
    const int j = ch * VC + lane;
    const bool active = j < p.nv;
    // v_j = -1 + (j + voff) dv, formed without contraction (vertex-centred variant PAPER.md:82-86)
    const double v = __dadd_rn(-1.0, __dmul_rn((double)j + p.voff, p.dv));
    const double wq = quad_weight(j, p.nv, p.quad);   // exactly 1 for the default Riemann sum
    mbar_wait(b_full_y + 8 * sy, (uint32_t)((n / NY) & 1));

    // ---- S2 (WENO7): right-interface fluxes of my rows, published for the neighbouring warp
    double FR[SCHEME == 1 ? S : 1][8];
    double nvz = 0.0, cadv_v = 0.0;
    if constexpr (SCHEME == 1) {
      nvz = v * p.ninv_dz;
      const cosenu_math::Weno7Beam bm = cosenu_math::weno7_beam(v, p.weno_eps);
      const uint32_t Tw = Ty + row0 * (VC * 8);
      const uint32_t Tc = Ty + (warp & 7) * (ROWS * VC * 8);   // boundary piece: component `warp` (warps 0..7)
      const unsigned mpos = __ballot_sync(0xffffffffu, v >= 0.0);
      const int xb = (int)(n % XBUF);                       // exchange buffer of this item
      const uint32_t xpar = (uint32_t)((n / XBUF) & 1);     // phase parity of its barriers
      // (a) my piece of the tile's left boundary flux first, so that warp 0 never waits for it
      if (warp < 8) {
        double FB;
        if (mpos == 0xffffffffu) FB = weno_boundary<1, ROWS, H>(Tc, bm);
        else if (mpos == 0u) FB = weno_boundary<-1, ROWS, H>(Tc, bm);
        else {
          const double bp = weno_boundary_slow<1, ROWS, H>(Tc, bm), bn = weno_boundary_slow<-1, ROWS, H>(Tc, bm);
          FB = v >= 0.0 ? bp : bn;
        }
        mbar_wait(b_xbr + 8 * xb, xpar ^ 1);   // warp 0 has read the previous contents
        sts(s_xb + xb * SM::XBSZ + (warp * VC + lane) * 8, FB);
        __syncwarp();
        if (lane == 0) mbar_arrive(b_xbf + 8 * xb);
      }
      // (b) the right-interface fluxes of my rows
      if (mpos == 0xffffffffu) {
        weno_rows<1, S, ROWS, H>(Tw, bm, FR);
      } else if (mpos == 0u) {
        weno_rows<-1, S, ROWS, H>(Tw, bm, FR);
      } else {
        double Fp[S * 8], Fm[S * 8];
        weno_rows_slow<1, S, ROWS, H>(Tw, bm, Fp);
        weno_rows_slow<-1, S, ROWS, H>(Tw, bm, Fm);
#pragma unroll
        for (int s = 0; s < S; ++s)
#pragma unroll
          for (int c = 0; c < 8; ++c) FR[s][c] = v >= 0.0 ? Fp[s * 8 + c] : Fm[s * 8 + c];
      }
      // (c) publish the flux of my last row for the warp that owns the next rows
      if (warp < NW - 1) {
        mbar_wait(b_xr + 8 * (xb * NSEG + warp), xpar ^ 1);   // it has read the previous contents
#pragma unroll
        for (int c = 0; c < 8; ++c) sts(s_x + xb * SM::XSZ + ((warp * 8 + c) * VC + lane) * 8, FR[S - 1][c]);
        __syncwarp();
        if (lane == 0) mbar_arrive(b_xf + 8 * (xb * NSEG + warp));
      }
    } else {
      cadv_v = v * p.cadv;
    }

    // broadcast helper: mu * moment q of my row s
    auto mom = [&](int s, int q) { return __shfl_sync(0xffffffffu, min_cur, s * 6 + q); };

    // rows in descending order: only row 0 needs the neighbour's flux, so its wait comes last
#pragma unroll
    for (int sd = 0; sd < S; ++sd) {
      const int s = S - 1 - sd;
      const int row = row0 + s;
      const long long iz = iz0 + row;
      const bool act = active && (iz < p.nz);
      const int tr = row + H;  // row inside the stage-input tile
      double yc[8], k[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) yc[c] = lds(Ty + ((c * ROWS + tr) * VC) * 8);

      // ---- S3: Hamiltonian from the moments (mu folded in), commutator
      {
        const double Sd = fma(-v, mom(s, 1), mom(s, 0));
        const double Sr = fma(-v, mom(s, 3), mom(s, 2));
        const double Si = fma(-v, mom(s, 5), mom(s, 4));
#pragma unroll
        for (int sp = 0; sp < 2; ++sp) {
          const double A = sp == 0 ? p.A0 + Sd : p.A0 - Sd;
          const double Br = sp == 0 ? p.Br0 + Sr : p.Br0 - Sr;
          const double Bi = Si;
          const int o = 4 * sp;
          const double dl = yc[o] - yc[o + 1];
          const double Tt = 2.0 * fma(Bi, yc[o + 2], -Br * yc[o + 3]);
          k[o] = Tt;
          k[o + 1] = -Tt;
          k[o + 2] = fma(A, yc[o + 3], -Bi * dl);
          k[o + 3] = fma(Br, dl, -A * yc[o + 2]);
        }
      }

      // ---- S2: advection
      if constexpr (SCHEME == 0) {
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          const uint32_t b = Ty + ((c * ROWS + tr) * VC) * 8;
          k[c] += cosenu_math::fd4_ko3(lds(b - 2 * VC * 8), lds(b - VC * 8), yc[c], lds(b + VC * 8), lds(b + 2 * VC * 8),
                                       cadv_v, p.cko);
        }
      } else if constexpr (SCHEME == 2) {
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          const uint32_t b = Ty + ((c * ROWS + tr) * VC) * 8;
          k[c] += cosenu_math::fd4_ko5(lds(b - 3 * VC * 8), lds(b - 2 * VC * 8), lds(b - VC * 8), yc[c], lds(b + VC * 8),
                                       lds(b + 2 * VC * 8), lds(b + 3 * VC * 8), cadv_v, p.cko);
        }
      } else {
        if (s == 0) {
          double FL[8];
          const int xb = (int)(n % XBUF);
          const uint32_t xpar = (uint32_t)((n / XBUF) & 1);
          if (warp == 0) {
            mbar_wait(b_xbf + 8 * xb, xpar);
#pragma unroll
            for (int c = 0; c < 8; ++c) FL[c] = lds(s_xb + xb * SM::XBSZ + (c * VC + lane) * 8);
            __syncwarp();
            if (lane == 0) mbar_arrive(b_xbr + 8 * xb);
          } else {
            mbar_wait(b_xf + 8 * (xb * NSEG + warp - 1), xpar);
#pragma unroll
            for (int c = 0; c < 8; ++c) FL[c] = lds(s_x + xb * SM::XSZ + (((warp - 1) * 8 + c) * VC + lane) * 8);
            __syncwarp();
            if (lane == 0) mbar_arrive(b_xr + 8 * (xb * NSEG + warp - 1));
          }
#pragma unroll
          for (int c = 0; c < 8; ++c) k[c] = fma(FR[0][c] - FL[c], nvz, k[c]);
        } else {
#pragma unroll
          for (int c = 0; c < 8; ++c) k[c] = fma(FR[s][c] - FR[s > 0 ? s - 1 : 0][c], nvz, k[c]);
        }
      }

      // ---- S4: RK combine; the outputs are staged in place in the u0/acc slot for the TMA store
      if (sd == 0) mbar_wait(b_full_ua + 8 * su, (uint32_t)((n / NUA) & 1));
      double out[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        const uint32_t cell = ((c * TZ + row) * VC) * 8;
        double u0v = yc[c], accb;
        if constexpr (KT::LOAD_U0) u0v = lds(Tu + cell);
        if constexpr (KIND == FIRST || KIND == FIRST_LEAN || KIND == MID_NOACC || KIND == MID_P) accb = yc[c];
        else if constexpr (KIND == MID_REBUILD) accb = fma(yc[c] - u0v, 1.0 / 3.0, u0v);  // u0 + (dt/6) k1
        else if constexpr (KIND == LAST_COMB) {
          // (Y2 + 2 Y3 + Y4 - U) / 3 = U + dt/6 (k1 + 2 k2 + 2 k3); Y4 is the stage input itself
          const double y2 = lds(Tu + SM::PTILE + cell), y3 = lds(Tu + 2 * SM::PTILE + cell);
          accb = (fma(2.0, y3, y2) + (yc[c] - u0v)) * (1.0 / 3.0);
        } else accb = lds(Ta_in + cell);
        // LAST_P: accb = P = (Y2 + 2 Y3 - U)/3 and the stage input is Y4: U+ = P + Y4/3 + dt/6 k4
        const double base = KIND == LAST_P ? fma(yc[c], 1.0 / 3.0, accb) : ((KIND == LAST || KIND == LAST_COMB) ? accb : u0v);
        const double o = fma(p.cy, k[c], base);
        sts(Tu + cell, o);
        if constexpr (KIND == MID_P) sts(Ta_out + cell, (fma(2.0, o, yc[c]) - u0v) * (1.0 / 3.0));   // P; yc = Y2, o = Y3
        else if constexpr (KT::WRITE_ACC) sts(Ta_out + cell, fma(p.ca, k[c], accb));
        out[c] = act ? o : 0.0;
      }
      // ghost copies of the first / last G rows of y_out are written directly: my own periodic ghost rows, or the
      // neighbouring slabs' ghost rows over NVLink (the halo exchange is fused into the producer)
      if (act && (iz < G || iz >= p.nz - G)) {
        if (iz < G) {
          double* d = p.ghost_lo_dst + iz * p.nvp + j;
#pragma unroll
          for (int c = 0; c < 8; ++c) d[c * p.ghost_lo_stride] = out[c];
        }
        if (iz >= p.nz - G) {
          double* d = p.ghost_hi_dst + (iz - (p.nz - G)) * p.nvp + j;
#pragma unroll
          for (int c = 0; c < 8; ++c) d[c * p.ghost_hi_stride] = out[c];
        }
      }

      // ---- S5: velocity moments of the produced state, D = rho - rhobar^*
      {
        double dd = (out[0] - out[1]) - (out[4] - out[5]), dr = out[2] - out[6], di = out[3] + out[7];
        if (p.quad != 0) { dd *= wq; dr *= wq; di *= wq; }   // uniform branch: the default rule costs no fp64 issue slots
        msum[6 * s + 0] += dd;
        msum[6 * s + 1] = fma(v, dd, msum[6 * s + 1]);
        msum[6 * s + 2] += dr;
        msum[6 * s + 3] = fma(v, dr, msum[6 * s + 3]);
        msum[6 * s + 4] += di;
        msum[6 * s + 5] = fma(v, di, msum[6 * s + 5]);
      }
    }

    // all reads of the stage-input slot are done, and my outputs are staged: tell the DMA warp
    fence_proxy_async();
    __syncwarp();
    if (lane == 0) {
      mbar_arrive(b_empty_y + 8 * sy);
      mbar_arrive(b_out_ready + 8 * su);
    }

    if (++ch == nchunks) {
      // end of the tile: reduce the partial moments over the lanes (fixed tree) and write them out
      int midx;
      bool mvalid;
      butterfly_reduce<6 * S>(msum, lane, midx, mvalid);
      if (mvalid) {
        const long long iz = iz0 + row0 + midx / 6;
        if (iz < p.nz) p.mom_out[(long long)(midx % 6) * p.nz + iz] = msum[0] * p.dv;
      }
#pragma unroll
      for (int q = 0; q < 6 * S; ++q) msum[q] = 0.0;
      // z-slab: tell the neighbours how many of their ghost rows this warp has just completed (all chunks)
      if (p.sig_lo != nullptr || p.sig_hi != nullptr) {
        int nlo = 0, nhi = 0;
#pragma unroll
        for (int s = 0; s < S; ++s) {
          const long long iz = iz0 + row0 + s;
          if (iz < p.nz) { nlo += iz < G; nhi += iz >= p.nz - G; }
        }
        if (nlo | nhi) {
          __threadfence_system();   // every lane: its ghost stores before the signal
          __syncwarp();
          if (lane == 0) {
            if (nlo && p.sig_lo != nullptr) red_add_release_sys(p.sig_lo, (unsigned long long)nlo);
            if (nhi && p.sig_hi != nullptr) red_add_release_sys(p.sig_hi, (unsigned long long)nhi);
          }
        }
      }
      ch = 0;
      ltile += gridDim.x;
    }
  }
}

}  // namespace cosenu_dev
