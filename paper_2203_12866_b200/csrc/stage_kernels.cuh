// stage_kernels.cuh -- ONE fused kernel per RK stage (sm_100a, fp64).
//
// Per launch and per (z,v) cell:
//   advection of the 8 real components by FD4+KO3 or FV-WENO7 (App. A),
//   Hamiltonian from the 6 per-z velocity moments of the stage input (Eq. 3a/3b),
//   commutator -i[H,rho], -i[Hbar,rhobar] (Eq. 1a/1b),
//   classical RK4 combine,
//   and, in the epilogue, the 6 velocity moments of the state just produced (the S1 of the next stage).
//
// Mapping.  Device layout of a state: double [8][nz + 2G][nvp], v fastest (G = 4 periodic ghost rows on
// each side of z, nvp = nv rounded up to 4).  One CTA owns TZ consecutive z rows and ALL v: it walks the
// v axis in chunks of VC beams.  The stage-input tile of a chunk ([8][TZ + 2H][VC] doubles, H = stencil
// halo) is brought into shared memory by ONE 3-D TMA box (cp.async.bulk.tensor) per chunk, double
// buffered on mbarriers, so the stencil reads come from shared memory and the load of chunk n+1
// overlaps the arithmetic of chunk n.  A thread = one beam (lane) x one z-segment of S = TZ/NSEG rows.
// u0 and the RK accumulator have no reuse and are read straight from global memory, coalesced over v.
// The moments are reduced over the lanes with shuffles and accumulated per row in shared memory in
// chunk order (fixed order => bit-reproducible; no atomics).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "weno7_math.h"

namespace cosenu_dev {

constexpr int G = 4;        // ghost rows per side in the device layout
constexpr int NBUF = 2;     // TMA double buffering

enum StageKind { FIRST = 0, FIRST_LEAN = 1, MID = 2, MID_REBUILD = 3, LAST = 4 };

struct StageParams {
  const double* u0;       // U (state at the beginning of the step), device layout; MID kinds only
  const double* acc_in;   // RK accumulator; MID and LAST
  double* y_out;          // next stage input (FIRST/MID) or the new U (LAST)
  double* acc_out;        // RK accumulator (FIRST, MID kinds)
  const double* mom_in;   // [6][nz] moments of the stage input (already times dv)
  double* mom_out;        // [6][nz] moments of y_out
  long long nz;
  int nv, nvp;
  long long comp_stride;  // (nz + 2G) * nvp
  double cy, ca;          // y_out = base + cy k ; acc_out = acc_in + ca k
  double mu, A0, Br0;     // A0 = -omega cos 2theta, Br0 = (omega/2) sin 2theta
  double dv;
  double cadv, cko;       // FD: -1/(12 dz), -eps_ko/(16 dz)   (times the advect switch)
  double ninv_dz, weno_eps;  // WENO: -1/dz (times the advect switch), epsilon of Eq. (14)
};

// ----------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// 3-D tiled TMA load global -> shared, completion on an mbarrier
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}

template <int SCHEME, int TZ, int VC>
struct StageSmem {
  static constexpr int H = SCHEME == 0 ? 2 : 4;
  static constexpr int ROWS = TZ + 2 * H;
  static constexpr int TILE = 8 * ROWS * VC;  // doubles per buffer
  static constexpr size_t bytes = sizeof(double) * ((size_t)NBUF * TILE + 12 * TZ) + 8 * NBUF + 128;
};

// ----------------------------------------------------------------------------- the stage kernel
template <int SCHEME, int KIND, int TZ, int NSEG, int VC>
__global__ void __launch_bounds__(NSEG* VC, 1)
    stage_kernel(const __grid_constant__ CUtensorMap tmap_y, const StageParams p) {
  using SM = StageSmem<SCHEME, TZ, VC>;
  constexpr int H = SM::H, ROWS = SM::ROWS, TILE = SM::TILE;
  constexpr int S = TZ / NSEG;
  constexpr int NT = NSEG * VC;
  constexpr bool LOAD_U0 = (KIND == MID || KIND == MID_REBUILD);
  constexpr bool LOAD_ACC = (KIND == MID || KIND == LAST);
  constexpr bool WRITE_ACC = (KIND == FIRST || KIND == MID || KIND == MID_REBUILD);
  static_assert(TZ % NSEG == 0 && VC <= 32 && (32 % VC) == 0, "tile shape");

  extern __shared__ unsigned char smem_raw[];
  double* tile = reinterpret_cast<double*>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~uintptr_t(127));
  double* s_min = tile + NBUF * TILE;   // [6][TZ]  mu * moments of the stage input
  double* s_macc = s_min + 6 * TZ;      // [6][TZ]  running moments of the output
  uint64_t* full = reinterpret_cast<uint64_t*>(s_macc + 6 * TZ);

  const int tid = threadIdx.x;
  const int lane = tid % VC;
  const int seg = tid / VC;
  const long long iz0 = (long long)blockIdx.x * TZ;
  const int nchunks = (p.nv + VC - 1) / VC;

  if (tid == 0) {
    for (int b = 0; b < NBUF; ++b) mbar_init(&full[b], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (int q = tid; q < 6 * TZ; q += NT) {
    const int m = q / TZ, r = q - m * TZ;
    const long long iz = iz0 + r;
    s_min[q] = iz < p.nz ? p.mu * p.mom_in[(long long)m * p.nz + iz] : 0.0;
    s_macc[q] = 0.0;
  }
  __syncthreads();
  if (tid == 0) {
    for (int b = 0; b < NBUF && b < nchunks; ++b) {
      mbar_expect_tx(&full[b], TILE * 8);
      tma_load_3d(tile + b * TILE, &tmap_y, &full[b], b * VC, (int)(iz0 + G - H), 0);
    }
  }

  for (int ch = 0; ch < nchunks; ++ch) {
    const int buf = ch % NBUF;
    const double* T = tile + buf * TILE;
    const int j = ch * VC + lane;
    const bool active = j < p.nv;
    // v_j = -1 + (j + 1/2) dv, formed without contraction
    const double v = __dadd_rn(-1.0, __dmul_rn((double)j + 0.5, p.dv));
    mbar_wait(&full[buf], (ch / NBUF) & 1);

    const int row0 = seg * S;
    double Fprev[8];
    int wdir = 1;
    double v2 = 0.0, nvz = 0.0, cadv_v = 0.0;
    if constexpr (SCHEME == 1) {
      wdir = v >= 0.0 ? 1 : -1;
      v2 = v * v;
      nvz = v * p.ninv_dz;
      // flux at the interface on the left of the segment's first cell
      const int rc = row0 - 1 + H + (wdir > 0 ? 0 : 1);
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        const double* b = T + (c * ROWS + rc) * VC + lane;
        double w[7];
#pragma unroll
        for (int k = 0; k < 7; ++k) w[k] = b[wdir * (k - 3) * VC];
        Fprev[c] = cosenu_math::weno7_face(w, v2, p.weno_eps);
      }
    } else {
      cadv_v = v * p.cadv;
    }

#pragma unroll 1
    for (int s = 0; s < S; ++s) {
      const int row = row0 + s;
      const long long iz = iz0 + row;
      const bool valid = iz < p.nz;      // ragged last tile: keep the lanes converged for the shuffles
      const bool act = active && valid;
      const int tr = row + H;  // row inside the tile
      double yc[8], k[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) yc[c] = T[(c * ROWS + tr) * VC + lane];

      // global operands with no reuse: issue early
      const long long gidx = (iz + G) * p.nvp + j;
      double u0v[8], accv[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        if constexpr (LOAD_U0) u0v[c] = act ? __ldg(p.u0 + c * p.comp_stride + gidx) : 0.0;
        else u0v[c] = yc[c];
        if constexpr (LOAD_ACC) accv[c] = act ? __ldg(p.acc_in + c * p.comp_stride + gidx) : 0.0;
      }

      // ---- S2: advection
      if constexpr (SCHEME == 0) {
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          const double* b = T + (c * ROWS + tr) * VC + lane;
          k[c] = cosenu_math::fd4_ko3(b[-2 * VC], b[-VC], yc[c], b[VC], b[2 * VC], cadv_v, p.cko);
        }
      } else {
        const int rc = tr + (wdir > 0 ? 0 : 1);
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          const double* b = T + (c * ROWS + rc) * VC + lane;
          double w[7];
#pragma unroll
          for (int q = 0; q < 7; ++q) w[q] = b[wdir * (q - 3) * VC];
          const double F = cosenu_math::weno7_face(w, v2, p.weno_eps);
          k[c] = (F - Fprev[c]) * nvz;
          Fprev[c] = F;
        }
      }

      // ---- S3: Hamiltonian from the moments (mu folded into s_min), commutator
      {
        const double Sd = fma(-v, s_min[1 * TZ + row], s_min[0 * TZ + row]);
        const double Sr = fma(-v, s_min[3 * TZ + row], s_min[2 * TZ + row]);
        const double Si = fma(-v, s_min[5 * TZ + row], s_min[4 * TZ + row]);
#pragma unroll
        for (int sp = 0; sp < 2; ++sp) {
          const double A = sp == 0 ? p.A0 + Sd : p.A0 - Sd;
          const double Br = sp == 0 ? p.Br0 + Sr : p.Br0 - Sr;
          const double Bi = Si;
          const int o = 4 * sp;
          const double dl = yc[o] - yc[o + 1];
          const double Tt = 2.0 * fma(Bi, yc[o + 2], -Br * yc[o + 3]);
          k[o] += Tt;
          k[o + 1] -= Tt;
          k[o + 2] += fma(A, yc[o + 3], -Bi * dl);
          k[o + 3] += fma(Br, dl, -A * yc[o + 2]);
        }
      }

      // ---- S4: RK combine and stores
      double out[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        double accb;
        if constexpr (KIND == FIRST || KIND == FIRST_LEAN) accb = yc[c];
        else if constexpr (KIND == MID_REBUILD) accb = fma(yc[c] - u0v[c], 1.0 / 3.0, u0v[c]);  // u0 + (dt/6) k1
        else accb = accv[c];
        const double base = (KIND == LAST) ? accb : u0v[c];
        out[c] = fma(p.cy, k[c], base);
        if (act) {
          double* yo = p.y_out + c * p.comp_stride + gidx;
          *yo = out[c];
          if (iz < G) yo[p.nz * p.nvp] = out[c];                 // right ghost copy of the first rows
          if (iz >= p.nz - G) yo[-p.nz * p.nvp] = out[c];        // left ghost copy of the last rows
          if constexpr (WRITE_ACC) p.acc_out[c * p.comp_stride + gidx] = fma(p.ca, k[c], accb);
        } else {
          out[c] = 0.0;
        }
      }

      // ---- S5: velocity moments of the produced state, D = rho - rhobar^*
      double m[6];
      m[0] = (out[0] - out[1]) - (out[4] - out[5]);
      m[2] = out[2] - out[6];
      m[4] = out[3] + out[7];
      m[1] = v * m[0];
      m[3] = v * m[2];
      m[5] = v * m[4];
#pragma unroll
      for (int q = 0; q < 6; ++q) {
#pragma unroll
        for (int off = VC / 2; off > 0; off >>= 1) m[q] += __shfl_xor_sync(0xffffffffu, m[q], off);
      }
      if (lane == 0 && valid) {
#pragma unroll
        for (int q = 0; q < 6; ++q) s_macc[q * TZ + row] += m[q];
      }
    }

    __syncthreads();  // every thread is done with this buffer
    if (tid == 0 && ch + NBUF < nchunks) {
      mbar_expect_tx(&full[buf], TILE * 8);
      tma_load_3d(tile + buf * TILE, &tmap_y, &full[buf], (ch + NBUF) * VC, (int)(iz0 + G - H), 0);
    }
  }

  __syncthreads();
  for (int q = tid; q < 6 * TZ; q += NT) {
    const int m = q / TZ, r = q - m * TZ;
    const long long iz = iz0 + r;
    if (iz < p.nz) p.mom_out[(long long)m * p.nz + iz] = s_macc[q] * p.dv;
  }
}

}  // namespace cosenu_dev
