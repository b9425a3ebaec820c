// aux_kernels.cuh -- kernels off the timed path: ghost rows, the moments of a freshly uploaded state,
// and the diagnostics reductions.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cosenu_dev {

// weight of beam j in the v' integral, in units of dv (int f dv ~ dv sum_j w_j f(v_j)):
//   quad 0: bin centres + Riemann sum -> 1;  on the vertex-centred grid of the FD variant
//   quad 1: trapezoid rule -> (1/2, 1, ..., 1, 1/2);  quad 2: Simpson's rule (nv odd) -> (1, 4, 2, ..., 4, 1)/3
__host__ __device__ __forceinline__ double quad_weight(int j, int nv, int quad) {
  if (quad == 0) return 1.0;
  const bool end = (j == 0) || (j == nv - 1);
  if (quad == 1) return end ? 0.5 : 1.0;
  return end ? 1.0 / 3.0 : ((j & 1) ? 4.0 / 3.0 : 2.0 / 3.0);
}

// periodic ghost rows of one state buffer: rows -G..-1 <- nz-G..nz-1, rows nz..nz+G-1 <- 0..G-1
__global__ void fill_ghosts_kernel(double* y, long long nz, int nvp, long long comp_stride, int g) {
  const long long n = (long long)8 * 2 * g * nvp;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < n; q += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(q % nvp);
    const int r = (int)((q / nvp) % (2 * g));
    const int c = (int)(q / ((long long)nvp * 2 * g));
    double* base = y + c * comp_stride;
    if (r < g) base[(long long)r * nvp + j] = base[(nz + r) * nvp + j];                  // device row r <- z = nz-g+r
    else base[(nz + r) * nvp + j] = base[(long long)r * nvp + j];                        // device row nz+r <- z = r-g
  }
}

// z-slab: copies of my first / last g rows of one state buffer into the neighbouring slabs' ghost rows (same
// destinations as the stage kernels use, see StageParams::ghost_*_dst); used once after an upload
__global__ void push_ghosts_kernel(const double* __restrict__ y, long long nz, int nvp, long long comp_stride, int g,
                                   double* dst_lo, long long stride_lo, double* dst_hi, long long stride_hi) {
  const long long n = (long long)8 * 2 * g * nvp;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < n; q += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(q % nvp);
    const int r = (int)((q / nvp) % (2 * g));
    const int c = (int)(q / ((long long)nvp * 2 * g));
    const double* src = y + c * comp_stride;
    if (r < g) dst_lo[c * stride_lo + (long long)r * nvp + j] = src[(long long)(g + r) * nvp + j];              // my row r
    else dst_hi[c * stride_hi + (long long)(r - g) * nvp + j] = src[(g + nz - g + (r - g)) * nvp + j];           // my row nz-g+(r-g)
  }
}

// cosenu_init on the device: the initial state is an outer product -- every entry is ONE product of a per-beam number
// (Eq. 20: g_nu(v_j), alpha g_nubar(v_j), normalised on the host) and a per-row number (the seeded phase or
// Eq. 21's Gaussian, evaluated on the host: O(nz + nv) libm calls in all).  The host uploads
// zv[4][nz] = (1 + d, 1 - d, Re, Im) and gv[2][nv] = (g, gbar) and this kernel forms the 8 planes, each entry with the same
// single rounding the host loop used to make ((g * 0.5) is exact), so the state is bit-identical to the old host expansion.
__global__ void init_expand_kernel(double* __restrict__ y, const double* __restrict__ zv, const double* __restrict__ gv,
                                   long long nz, int nv, int nvp, long long comp_stride, int g) {
  for (long long iz = blockIdx.x; iz < nz; iz += gridDim.x) {
    const double ap = zv[iz], am = zv[nz + iz], pr = zv[2 * nz + iz], pi = zv[3 * nz + iz];
    double* row = y + (iz + g) * nvp;
    for (int j = threadIdx.x; j < nv; j += blockDim.x) {
      const double gj = gv[j], gbj = gv[nv + j];
      const double hg = __dmul_rn(gj, 0.5), hgb = __dmul_rn(gbj, 0.5);
      row[j] = __dmul_rn(hg, ap);                     row[comp_stride + j] = __dmul_rn(hg, am);
      row[2 * comp_stride + j] = __dmul_rn(gj, pr);   row[3 * comp_stride + j] = __dmul_rn(gj, pi);
      row[4 * comp_stride + j] = __dmul_rn(hgb, ap);  row[5 * comp_stride + j] = __dmul_rn(hgb, am);
      row[6 * comp_stride + j] = __dmul_rn(gbj, pr);  row[7 * comp_stride + j] = __dmul_rn(gbj, pi);
    }
  }
}

// the 6 velocity moments per z of a state (S1; Riemann sum of PAPER.md:78): one warp per z row,
// lanes stride over v, fixed shuffle tree => reproducible.  mom[6][nz], already times dv.
__global__ void moments_kernel(const double* __restrict__ y, double* __restrict__ mom, long long nz, int nv, int nvp,
                               long long comp_stride, int g, double dv, double voff, int quad) {
  const int warps = blockDim.x / 32, wid = threadIdx.x / 32, lane = threadIdx.x % 32;
  for (long long iz = blockIdx.x * (long long)warps + wid; iz < nz; iz += (long long)gridDim.x * warps) {
    double m[6] = {0, 0, 0, 0, 0, 0};
    const double* row = y + (iz + g) * nvp;
    for (int j = lane; j < nv; j += 32) {
      const double v = __dadd_rn(-1.0, __dmul_rn((double)j + voff, dv));
      const double wq = quad_weight(j, nv, quad);
      const double dd = wq * ((row[j] - row[comp_stride + j]) - (row[4 * comp_stride + j] - row[5 * comp_stride + j]));
      const double dr = wq * (row[2 * comp_stride + j] - row[6 * comp_stride + j]);
      const double di = wq * (row[3 * comp_stride + j] + row[7 * comp_stride + j]);
      m[0] += dd; m[1] = fma(v, dd, m[1]);
      m[2] += dr; m[3] = fma(v, dr, m[3]);
      m[4] += di; m[5] = fma(v, di, m[5]);
    }
#pragma unroll
    for (int q = 0; q < 6; ++q) {
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) m[q] += __shfl_xor_sync(0xffffffffu, m[q], off);
      if (lane == 0) mom[(long long)q * nz + iz] = m[q] * dv;
    }
  }
}

__device__ __forceinline__ double plen(double ee, double xx, double r, double i) {
  const double d = ee - xx;
  return sqrt(fma(d, d, 4.0 * fma(r, r, i * i)));  // |P| of Eq. (4), un-normalised
}

// z-slab partial sums of |P|(z,v) and P0(z,v) per species: part[b][4][nv] (|P|_nu, P0_nu, |P|_nubar, P0_nubar).
// blockDim = DIAG_REF_ROWS x DIAG_REF_LANES: lane = beam (coalesced rows), DIAG_REF_ROWS rows of the block's z-range in flight
// at once and two rows per thread and trip, so that the reads of a block cover the HBM latency; the row groups are summed
// in a fixed order (reproducible).
constexpr int DIAG_REF_ROWS = 4, DIAG_REF_LANES = 256;
__global__ void __launch_bounds__(DIAG_REF_ROWS * DIAG_REF_LANES)
    diag_ref_kernel(const double* __restrict__ y, double* __restrict__ part, long long nz, int nv, int nvp,
                    long long comp_stride, int g) {
  __shared__ double red[DIAG_REF_ROWS][4][DIAG_REF_LANES];
  const int tj = threadIdx.x % DIAG_REF_LANES, tr = threadIdx.x / DIAG_REF_LANES;
  const long long rows_per = (nz + gridDim.x - 1) / gridDim.x;
  const long long z0 = blockIdx.x * rows_per, z1 = min(nz, z0 + rows_per);
  for (int j0 = 0; j0 < nv; j0 += DIAG_REF_LANES) {
    const int j = j0 + tj;
    double a[4] = {0, 0, 0, 0}, b[4] = {0, 0, 0, 0};
    if (j < nv) {
      auto row = [&](long long iz, double (&acc)[4]) {
        const double* q = y + (iz + g) * nvp + j;
        double c[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) c[k] = q[k * comp_stride];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
          acc[2 * s] += plen(c[4 * s], c[4 * s + 1], c[4 * s + 2], c[4 * s + 3]);
          acc[2 * s + 1] += c[4 * s] + c[4 * s + 1];
        }
      };
      long long iz = z0 + tr;
      for (; iz + DIAG_REF_ROWS < z1; iz += 2 * DIAG_REF_ROWS) { row(iz, a); row(iz + DIAG_REF_ROWS, b); }
      if (iz < z1) row(iz, a);
    }
#pragma unroll
    for (int m = 0; m < 4; ++m) red[tr][m][tj] = a[m] + b[m];
    __syncthreads();
    if (tr == 0 && j < nv) {
#pragma unroll
      for (int m = 0; m < 4; ++m) {
        double sum = red[0][m][tj];
#pragma unroll
        for (int r = 1; r < DIAG_REF_ROWS; ++r) sum += red[r][m][tj];
        part[((long long)blockIdx.x * 4 + m) * nv + j] = sum;
      }
    }
    __syncthreads();
  }
}

constexpr int DIAG_NSUM = 7;  // see_nu, see_nubar, sum| |P_nu| - Pref |, M0x, M0y, M0z, (spare)
constexpr int DIAG_NMAX = 3;  // dP_max, trace_dev_max, ex_abs_max
constexpr int DIAG_NVAL = DIAG_NSUM + DIAG_NMAX;

// per-block partial diagnostics over a z-slab: part[b][DIAG_NVAL]
__global__ void diag_kernel(const double* __restrict__ y, const double* __restrict__ pref /*[2][nv]*/,
                            const double* __restrict__ p0ref /*[2][nv]*/, double* __restrict__ part, long long nz,
                            int nv, int nvp, long long comp_stride, int g, int quad) {
  const long long rows_per = (nz + gridDim.x - 1) / gridDim.x;
  const long long z0 = blockIdx.x * rows_per, z1 = min(nz, z0 + rows_per);
  double sm[DIAG_NSUM] = {0, 0, 0, 0, 0, 0, 0};
  double mx[DIAG_NMAX] = {0, 0, 0};
  for (int j = threadIdx.x; j < nv; j += blockDim.x) {
    const double pr[2] = {pref[j], pref[nv + j]}, p0[2] = {p0ref[j], p0ref[nv + j]};
    const double wq = quad_weight(j, nv, quad);   // the v-sums of PAPER.md:229, Eq. (19), Eq. (23) use the rule of the v' integral
    for (long long iz = z0; iz < z1; ++iz) {
      const double* q = y + (iz + g) * nvp + j;
      double c[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) c[k] = q[k * comp_stride];
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        const double ee = c[4 * s], xx = c[4 * s + 1], r = c[4 * s + 2], im = c[4 * s + 3];
        sm[s] += wq * ee;
        const double P = plen(ee, xx, r, im);
        if (pr[s] > 0) mx[0] = fmax(mx[0], fabs(P / pr[s] - 1.0));   // Eq. (22)
        if (s == 0) sm[2] += wq * fabs(P - pr[0]);                       // numerator of Eq. (23)
        mx[1] = fmax(mx[1], fabs(ee + xx - p0[s]));
        mx[2] = fmax(mx[2], sqrt(fma(r, r, im * im)));
      }
      // Eq. (19) in stored variables: P = (2 Re, -2 Im, ee - xx) of D = rho - rhobar^*
      sm[3] += wq * (2.0 * (c[2] - c[6]));
      sm[4] += wq * (-2.0 * (c[3] + c[7]));
      sm[5] += wq * ((c[0] - c[1]) - (c[4] - c[5]));
    }
  }
  __shared__ double red[32][DIAG_NVAL];
  const int lane = threadIdx.x % 32, wid = threadIdx.x / 32, nw = blockDim.x / 32;
#pragma unroll
  for (int k = 0; k < DIAG_NSUM; ++k)
    for (int off = 16; off > 0; off >>= 1) sm[k] += __shfl_xor_sync(0xffffffffu, sm[k], off);
#pragma unroll
  for (int k = 0; k < DIAG_NMAX; ++k)
    for (int off = 16; off > 0; off >>= 1) mx[k] = fmax(mx[k], __shfl_xor_sync(0xffffffffu, mx[k], off));
  if (lane == 0) {
    for (int k = 0; k < DIAG_NSUM; ++k) red[wid][k] = sm[k];
    for (int k = 0; k < DIAG_NMAX; ++k) red[wid][DIAG_NSUM + k] = mx[k];
  }
  __syncthreads();
  if (threadIdx.x < DIAG_NVAL) {
    const int k = threadIdx.x;
    double a = red[0][k];
    for (int w = 1; w < nw; ++w) a = k < DIAG_NSUM ? a + red[w][k] : fmax(a, red[w][k]);
    part[(long long)blockIdx.x * DIAG_NVAL + k] = a;
  }
}

}  // namespace cosenu_dev
