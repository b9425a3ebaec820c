// weno_march.cuh -- the FV-WENO7 stage kernel of the default RK carrier (sm_100a, fp64): one fused, persistent,
// role-specialised kernel per RK stage.
//
// Same work per launch and per (z,v) cell as stage_kernel<1, ...> (stage_kernels.cuh): WENO7 advection with v-sign
// upwinding (App. A / Algorithm 1), Hamiltonian from the 6 per-z moments and commutator
// (Eqs. 1-3), classical RK4 combine, moments of the produced state.  Same arithmetic per cell
// (weno7_math.h), so the results are bit-identical to stage_kernel's; what differs is who computes what:
//
//  * The reconstruction is independent per real component and is 90 % of the fp64 work.  WENO warp c (c = 0..7) owns
//    component c of a work item (z-tile of TZ = 16 rows x chunk of 32 beams, lane = beam) and MARCHES along z through the
//    tile: every cell is read from shared memory once, every undivided difference D, E, T and T^2 of Algorithm 1 is
//    formed once and slides through registers, every interface value is computed once (TZ + 1 per march; the first one
//    is the only recomputation, 1/16).  No flux is exchanged between warps.  Two marches run interleaved in one thread
//    -- from the low end of the tile upwards and from the high end downwards, meeting in the middle -- which gives the
//    scheduler two independent dependency chains per warp (DFMA latency 8 clk, issue 1 per 2 clk and sub-partition).
//    For v < 0 the same code marches through the mirrored tile (reading A9 of DESIGN.md).  The flux differences
//    F_{i+1/2} - F_{i-1/2} go to shared memory.
//  * Four COMBINE warps (4 rows each) read the cell values, the flux differences and the RK operands, form the
//    commutator, the RK combination and the moments, and stage the outputs for the TMA store.  They run one item behind
//    the WENO warps, so the load/store-heavy and the fp64-dense phases overlap by construction instead of by chance.
//  * One DMA lane feeds the rings with 3-D TMA boxes and issues the TMA stores, as in stage_kernel.
//
// Shared memory (224 KB): 2 stage-input slots [8][24][32] + 2 operand slots of two arrays [8][16][32]: A0 = u0 / P on load,
// y_out on store; A1 = flux differences, then P on store (stage 2).
#pragma once
#include "stage_kernels.cuh"

namespace cosenu_dev {

constexpr int MTZ = 16;                 // rows per tile
constexpr int MROWS = MTZ + 2 * G;      // with the WENO halo of 4
constexpr int MNW = 8, MNC = 4;         // WENO warps (one per component), combine warps
constexpr int MRC = MTZ / MNC;          // rows per combine warp
constexpr int MARCH_THREADS = (MNW + MNC + 4) * 32;   // + the DMA warp and three idle warps (a full warpgroup for setmaxnreg)
// registers per thread after the roles have split (the kernel is launched with 512 threads x 128 registers; every SM
// sub-partition holds two WENO warps, one combine warp and one warp of the DMA group): 2 x 160 + 152 + 40 = 512
constexpr int MREG_WENO = 160, MREG_COMB = 152, MREG_DMA = 40;

struct MarchSmem {
  static constexpr uint32_t YTILE = 8u * MROWS * VC * 8u;
  static constexpr uint32_t PTILE = 8u * MTZ * VC * 8u;
  static constexpr uint32_t off_y = 0;                    // [2][YTILE]
  static constexpr uint32_t off_a = 2 * YTILE;            // [2][2][PTILE]
  static constexpr uint32_t off_bar = off_a + 4 * PTILE;  // full_y[2] empty_y[2] full_a[2] a_free[2] k_ready[2] out_ready[2]
  static constexpr size_t bytes = off_bar + 8 * 12 + 128;
};

// one march of one component through the tile.  Ty0 / Tk0: shared addresses of (component, row 0, this lane) of the
// stage-input slot (halo included) and of the flux-difference array.
// March coordinates: cell j = 0..22 is tile row j (DIR > 0) or 23 - j (DIR < 0); interface m = 0..16 lies between cells
// m + 3 and m + 4 and is biased towards smaller j (the upwind side); march row r' = 0..15 is cell r' + 4 and gets
// F[r' + 1] - F[r'], stored at real row r' (DIR > 0) or 15 - r' (DIR < 0).  DIR == 0: per-lane direction (`neg`).
// The first flux difference is stored after the second interface: only then must the flux-difference array of the slot be
// free (barrier `bar_free`, phase parity `par_free`), so that wait hides behind the first two interfaces.
template <int DIR>
__device__ __forceinline__ void weno_march(uint32_t Ty0, uint32_t Tk0, bool neg, const cosenu_math::Weno7Beam& bm,
                                           uint32_t bar_free, uint32_t par_free) {
  constexpr int RB = VC * 8;   // bytes per row
  uint32_t yb = Ty0, kb = Tk0;
  int ys = RB;
  if constexpr (DIR == 0) {
    yb = neg ? Ty0 + (MROWS - 1) * RB : Ty0;
    kb = neg ? Tk0 + (MTZ - 1) * RB : Tk0;
    ys = neg ? -RB : RB;
  }
  auto cell = [&](int j) -> double {
    if constexpr (DIR > 0) return lds(Ty0 + j * RB);
    else if constexpr (DIR < 0) return lds(Ty0 + (MROWS - 1 - j) * RB);
    else return lds(yb + j * ys);
  };
  auto put = [&](int r, double x) {
    if constexpr (DIR > 0) sts(Tk0 + r * RB, x);
    else if constexpr (DIR < 0) sts(Tk0 + (MTZ - 1 - r) * RB, x);
    else sts(kb + r * ys, x);
  };
  constexpr int NI = MTZ + 1;        // interfaces 0..16
  constexpr int NLO = (NI + 1) / 2;  // the upward march takes m = 0..8, the downward one m = 16..9
  double c[MROWS - 1], D[MROWS - 2], E[MROWS - 3], T[MROWS - 4], TT[MROWS - 4];
  // start of the upward march: cells 0..5; of the downward one: cells 17..22
#pragma unroll
  for (int j = 0; j < 6; ++j) c[j] = cell(j);
#pragma unroll
  for (int j = MROWS - 7; j < MROWS - 1; ++j) c[j] = cell(j);
#pragma unroll
  for (int j = 0; j < 5; ++j) D[j] = c[j + 1] - c[j];
#pragma unroll
  for (int j = MROWS - 7; j < MROWS - 2; ++j) D[j] = c[j + 1] - c[j];
#pragma unroll
  for (int j = 0; j < 4; ++j) E[j] = D[j + 1] - D[j];
#pragma unroll
  for (int j = MROWS - 7; j < MROWS - 3; ++j) E[j] = D[j + 1] - D[j];
#pragma unroll
  for (int j = 0; j < 3; ++j) { T[j] = E[j + 1] - E[j]; TT[j] = T[j] * T[j]; }
#pragma unroll
  for (int j = MROWS - 7; j < MROWS - 4; ++j) { T[j] = E[j + 1] - E[j]; TT[j] = T[j] * T[j]; }
  double Flo = 0.0, Fhi = 0.0;
  // X[idx] (X = c, D, E, T) is needed by the upward march at step idx - (6, 5, 4, 3) and by the downward one at step
  // NI - 1 - idx; whichever comes first (the upward march goes first within a step) forms it, once.
  // The shared-memory loads are issued PD steps ahead of their use: a load cannot pass an earlier store to shared memory (the
  // flux differences of the previous interfaces), so a load issued where its cell is first needed would wait for the end of the
  // previous interface's dependency chain and serialise the two marches.
  constexpr int PD = 2;
  auto up_loads = [&](int s) {     // the cell the upward march needs at step s, if it is the upward march's to load
    if (s < NLO && 2 * s + 6 <= NI - 1) c[s + 6] = cell(s + 6);
  };
  auto down_loads = [&](int s) {   // likewise for the downward march (interface m = NI - 1 - s, new cell m)
    if (s < NI - NLO && (NI - 1 - s) - 6 > s) c[NI - 1 - s] = cell(NI - 1 - s);
  };
#pragma unroll
  for (int s = 0; s < PD; ++s) { up_loads(s); down_loads(s); }
#pragma unroll
  for (int s = 0; s < NLO; ++s) {
    if (s == 1) mbar_wait(bar_free, par_free);
    up_loads(s + PD);
    down_loads(s + PD);
    {   // upward march, interface m = s: the new cell is m + 6
      const int m = s;
      if (2 * s + 5 <= NI - 1) D[m + 5] = c[m + 6] - c[m + 5];
      if (2 * s + 4 <= NI - 1) E[m + 4] = D[m + 5] - D[m + 4];
      if (2 * s + 3 <= NI - 1) { T[m + 3] = E[m + 4] - E[m + 3]; TT[m + 3] = T[m + 3] * T[m + 3]; }
      const double F = cosenu_math::weno7_core(c[m + 3], D[m], D[m + 1], D[m + 2], D[m + 3], E[m], E[m + 1], E[m + 2],
                                               E[m + 3], E[m + 4], T[m], T[m + 3], TT[m], TT[m + 1], TT[m + 2], TT[m + 3], bm);
      if (m >= 1) put(m - 1, F - Flo);
      Flo = F;
    }
    if (s < NI - NLO) {   // downward march, interface m = NI - 1 - s: the new cell is m
      const int m = NI - 1 - s;
      if (m - 5 > s) D[m] = c[m + 1] - c[m];
      if (m - 4 > s) E[m] = D[m + 1] - D[m];
      if (m - 3 > s) { T[m] = E[m + 1] - E[m]; TT[m] = T[m] * T[m]; }
      const double F = cosenu_math::weno7_core(c[m + 3], D[m], D[m + 1], D[m + 2], D[m + 3], E[m], E[m + 1], E[m + 2],
                                               E[m + 3], E[m + 4], T[m], T[m + 3], TT[m], TT[m + 1], TT[m + 2], TT[m + 3], bm);
      if (m <= NI - 2) put(m, Fhi - F);
      Fhi = F;
    }
  }
  put(NLO - 1, Fhi - Flo);   // the row between the last interfaces of the two marches
}

template <int KIND>
__global__ void __launch_bounds__(MARCH_THREADS, 1)
    weno_march_kernel(const __grid_constant__ CUtensorMap tm_y,     // stage input with halo: box [8][24][32]
                      const __grid_constant__ CUtensorMap tm_u0,    // U, rows 0..nz-1: box [8][16][32]
                      const __grid_constant__ CUtensorMap tm_acc,   // P (stored by stage 2, loaded by stage 4)
                      const __grid_constant__ CUtensorMap tm_out,   // y_out, rows 0..nz-1
                      const StageParams p) {
  using SM = MarchSmem;
  using KT = KindTraits<KIND>;
  static_assert(KIND == FIRST_LEAN || KIND == MID_P || KIND == MID_NOACC || KIND == LAST_P, "kinds of the partial-sum RK carrier");
  static_assert(KT::NLOAD <= 1, "one loaded operand array");
  constexpr int TZ = MTZ, ROWS = MROWS, H = G;

  extern __shared__ unsigned char smem_raw[];
  const uint32_t sbase = (smem_u32(smem_raw) + 127u) & ~127u;
  const uint32_t s_y = sbase + SM::off_y, s_a = sbase + SM::off_a, s_bar = sbase + SM::off_bar;
  const uint32_t b_full_y = s_bar, b_empty_y = s_bar + 16, b_full_a = s_bar + 32, b_a_free = s_bar + 48,
                 b_k_ready = s_bar + 64, b_out_ready = s_bar + 80;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nchunks = (p.nv + VC - 1) / VC;
  const long long ntiles = (p.nz + TZ - 1) / TZ;
  const long long my_tiles = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const int nitems = (int)(my_tiles * nchunks);   // items of this CTA (fits: at most nz / 16 / gridDim.x * nv / 32)
  auto tile_of = [&](long long l) { const long long t = l + p.tile_shift; return t >= ntiles ? t - ntiles : t; };

  if (threadIdx.x == 0) {
    for (int b = 0; b < 2; ++b) {
      mbar_init(b_full_y + 8 * b, 1); mbar_init(b_empty_y + 8 * b, MNW + MNC);
      mbar_init(b_full_a + 8 * b, 1); mbar_init(b_a_free + 8 * b, 1);
      mbar_init(b_k_ready + 8 * b, MNW); mbar_init(b_out_ready + 8 * b, MNC);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // =========================================================================== DMA warp (one lane)
  if (warp >= MNW + MNC) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(MREG_DMA));
    if (warp == MNW + MNC && lane == 0) {
      auto store_item = [&](int m) {
        const int su = (int)(m & 1);
        const int iz0 = (int)(tile_of(blockIdx.x + (m / nchunks) * gridDim.x) * TZ), c0 = (int)(m % nchunks) * VC;
        mbar_wait(b_out_ready + 8 * su, (uint32_t)((m >> 1) & 1));
        const uint32_t src = s_a + su * 2 * SM::PTILE;
        tma_store_3d(&tm_out, src, c0, iz0, 0);
        if constexpr (KT::WRITE_ACC) tma_store_3d(&tm_acc, src + SM::PTILE, c0, iz0, 0);
        tma_store_commit();
        tma_store_wait_read();   // both arrays of the slot may be overwritten from here on
      };
      long long ltile = blockIdx.x;
      int ch = 0;
      for (int n = 0; n < nitems; ++n) {
        const long long tile = tile_of(ltile);
        const int iz0 = (int)(tile * TZ);
        const int sy = (int)(n & 1), su = sy;
        if (ch == 0 && (p.wait_lo != nullptr || p.wait_hi != nullptr)) {
          bool waited = false;
          if (p.wait_lo != nullptr && tile * TZ < G) { wait_arrivals(p.wait_lo, p.wait_val, p.err_flag, p.wait_timeout_ns); waited = true; }
          if (p.wait_hi != nullptr && (tile + 1) * TZ + G > p.nz) { wait_arrivals(p.wait_hi, p.wait_val, p.err_flag, p.wait_timeout_ns); waited = true; }
          if (waited) asm volatile("fence.proxy.async.global;" ::: "memory");
        }
        mbar_wait(b_empty_y + 8 * sy, (uint32_t)(((n >> 1) & 1) ^ 1));
        mbar_expect_tx(b_full_y + 8 * sy, SM::YTILE);
        tma_load_3d(s_y + sy * SM::YTILE, &tm_y, b_full_y + 8 * sy, ch * VC, iz0 + G - H, 0);
        if (n >= 2) store_item(n - 2);
        mbar_arrive(b_a_free + 8 * su);   // the WENO warps may write their flux differences into A1 of this slot
        if constexpr (KT::NLOAD > 0) {
          mbar_expect_tx(b_full_a + 8 * su, SM::PTILE);
          tma_load_3d(s_a + su * 2 * SM::PTILE, KT::LOAD_U0 ? &tm_u0 : &tm_acc, b_full_a + 8 * su, ch * VC, iz0, 0);
        } else {
          mbar_arrive(b_full_a + 8 * su);
        }
        if (++ch == nchunks) { ch = 0; ltile += gridDim.x; }
      }
      for (int m = nitems > 2 ? nitems - 2 : 0; m < nitems; ++m) store_item(m);
      tma_store_wait_all();
    }
    return;
  }

  // =========================================================================== WENO warps: component `warp`
  if (warp < MNW) {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(MREG_WENO));
    int ch = 0;
    for (int n = 0; n < nitems; ++n) {
      const int sy = (int)(n & 1), su = sy;
      const uint32_t par = (uint32_t)((n >> 1) & 1);
      const int j = ch * VC + lane;
      const double v = __dadd_rn(-1.0, __dmul_rn((double)j + p.voff, p.dv));
      const cosenu_math::Weno7Beam bm = cosenu_math::weno7_beam(v, p.weno_eps);
      const unsigned mpos = __ballot_sync(0xffffffffu, v >= 0.0);
      const uint32_t Ty0 = s_y + sy * SM::YTILE + (warp * ROWS * VC + lane) * 8;
      const uint32_t Tk0 = s_a + (su * 2 + 1) * SM::PTILE + (warp * TZ * VC + lane) * 8;
      mbar_wait(b_full_y + 8 * sy, par);
      if (mpos == 0xffffffffu) weno_march<1>(Ty0, Tk0, false, bm, b_a_free + 8 * su, par);
      else if (mpos == 0u) weno_march<-1>(Ty0, Tk0, true, bm, b_a_free + 8 * su, par);
      else weno_march<0>(Ty0, Tk0, v < 0.0, bm, b_a_free + 8 * su, par);
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(b_empty_y + 8 * sy);
        mbar_arrive(b_k_ready + 8 * su);
      }
      if (++ch == nchunks) ch = 0;
    }
    return;
  }

  // =========================================================================== combine warps: rows 4q .. 4q+3
  asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(MREG_COMB));
  const int q = warp - MNW;
  const int row0 = q * MRC;
  double msum[6 * MRC];
#pragma unroll
  for (int i = 0; i < 6 * MRC; ++i) msum[i] = 0.0;
  auto load_min = [&](long long l) {
    double m = 0.0;
    if (lane < 6 * MRC && l < ntiles) {
      const long long iz = tile_of(l) * TZ + row0 + lane / 6;
      if (iz < p.nz) m = __ldg(p.mom_in + (long long)(lane % 6) * p.nz + iz);
    }
    return m;
  };
  double min_cur = 0.0, min_next = load_min(blockIdx.x);
  long long ltile = blockIdx.x;
  int ch = 0;
  for (int n = 0; n < nitems; ++n) {
    const long long iz0 = tile_of(ltile) * TZ;
    if (ch == 0) {
      min_cur = p.mu * min_next;
      min_next = load_min(ltile + gridDim.x);
    }
    const int sy = (int)(n & 1), su = sy;
    const uint32_t par = (uint32_t)((n >> 1) & 1);
    const uint32_t Ty = s_y + sy * SM::YTILE + lane * 8;              // + ((c * ROWS + r) * 32) * 8
    const uint32_t Tu = s_a + su * 2 * SM::PTILE + lane * 8;          // + ((c * TZ + r) * 32) * 8
    const uint32_t Tk = Tu + SM::PTILE;
    const int j = ch * VC + lane;
    const bool active = j < p.nv;
    const double v = __dadd_rn(-1.0, __dmul_rn((double)j + p.voff, p.dv));
    const double wq = quad_weight(j, p.nv, p.quad);
    const double cf = fabs(v) * p.ninv_dz;   // -|v|/dz: the flux differences are taken along the march (upwind to downwind)
    auto mom = [&](int s, int qq) { return __shfl_sync(0xffffffffu, min_cur, s * 6 + qq); };

    // the cell values of my rows are read as soon as the stage-input tile is there -- while the WENO warps still march through
    // it -- and the slot is released at once: it is then free the moment the marches end, and the TMA load of the item after
    // next has a whole item time (one SM's share of HBM needs 1.1 us for a tile, an item takes 2.5-3 us)
    mbar_wait(b_full_y + 8 * sy, par);
    double yca[MRC][8];
#pragma unroll
    for (int s = 0; s < MRC; ++s)
#pragma unroll
      for (int c = 0; c < 8; ++c) yca[s][c] = lds(Ty + ((c * ROWS + row0 + s + H) * VC) * 8);
    __syncwarp();
    if (lane == 0) mbar_arrive(b_empty_y + 8 * sy);
    mbar_wait(b_k_ready + 8 * su, par);
    mbar_wait(b_full_a + 8 * su, par);
#pragma unroll
    for (int s = 0; s < MRC; ++s) {
      const int row = row0 + s;
      const long long iz = iz0 + row;
      const bool act = active && (iz < p.nz);
      double yc[8], k[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) yc[c] = yca[s][c];
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
      // ---- S2: advection from the flux differences of the WENO warps;  S4: RK combine, staged in place
      double out[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        const uint32_t cell = ((c * TZ + row) * VC) * 8;
        k[c] = fma(lds(Tk + cell), cf, k[c]);
        double u0v = yc[c], accb = yc[c];
        if constexpr (KT::LOAD_U0) u0v = lds(Tu + cell);
        if constexpr (KIND == LAST_P) accb = lds(Tu + cell);   // P = (Y2 + 2 Y3 - U)/3; the stage input is Y4
        const double base = KIND == LAST_P ? fma(yc[c], 1.0 / 3.0, accb) : u0v;
        const double o = fma(p.cy, k[c], base);
        sts(Tu + cell, o);
        if constexpr (KIND == MID_P) sts(Tk + cell, (fma(2.0, o, yc[c]) - u0v) * (1.0 / 3.0));   // P; yc = Y2, o = Y3
        out[c] = o;
      }
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
        if (!act) { dd = 0.0; dr = 0.0; di = 0.0; }   // padding lanes / rows past the grid hold zero-filled cells: no contribution
        if (p.quad != 0) { dd *= wq; dr *= wq; di *= wq; }
        msum[6 * s + 0] += dd;
        msum[6 * s + 1] = fma(v, dd, msum[6 * s + 1]);
        msum[6 * s + 2] += dr;
        msum[6 * s + 3] = fma(v, dr, msum[6 * s + 3]);
        msum[6 * s + 4] += di;
        msum[6 * s + 5] = fma(v, di, msum[6 * s + 5]);
      }
    }
    fence_proxy_async();
    __syncwarp();
    if (lane == 0) mbar_arrive(b_out_ready + 8 * su);

    if (++ch == nchunks) {
      int midx;
      bool mvalid;
      butterfly_reduce<6 * MRC>(msum, lane, midx, mvalid);
      if (mvalid) {
        const long long iz = iz0 + row0 + midx / 6;
        if (iz < p.nz) p.mom_out[(long long)(midx % 6) * p.nz + iz] = msum[0] * p.dv;
      }
#pragma unroll
      for (int i = 0; i < 6 * MRC; ++i) msum[i] = 0.0;
      if (p.sig_lo != nullptr || p.sig_hi != nullptr) {
        int nlo = 0, nhi = 0;
#pragma unroll
        for (int s = 0; s < MRC; ++s) {
          const long long iz = iz0 + row0 + s;
          if (iz < p.nz) { nlo += iz < G; nhi += iz >= p.nz - G; }
        }
        if (nlo | nhi) {
          __threadfence_system();
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
