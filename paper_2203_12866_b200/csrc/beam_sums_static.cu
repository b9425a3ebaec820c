// beam_sums_static.cu -- cosenu_beam_sums_static (include/cosenu.h): the per-beam z-sums of |P| and P0 of both species
// (Eq. 4; they become the t = 0 references of Eq. 22, 23) for callers that must not
// allocate device memory.
//
// The handle-based route to these numbers (diag_ref_kernel in aux_kernels.cuh, reached through cosenu_slab_ref_sums) keeps its
// per-block partial sums in the handle's workspace, and a workspace has to be allocated by somebody.  Here the partial sums
// live in a fixed array that is part of the library image instead, so this one call needs no cudaMalloc, no cudaFree, no
// stream-ordered allocation and no handle: inputs and outputs are the caller's device buffers, and that is all the memory
// the call touches apart from the array below.
//
// This is its own translation unit on purpose: the array has internal linkage, and the address the kernels need is looked
// up (cudaGetSymbolAddress) by host code of this same file.  It shares no kernel with cosenu_api.cu; the existing paths are
// untouched.
#include "../../include/cosenu.h"

#include <cuda_runtime.h>

#include <mutex>
#include <string>

namespace {

constexpr int SB_BLOCKS = 148;              // z-ranges, i.e. partial sums per (quantity, beam); fixed, so that results do not depend on the GPU
constexpr int SB_ROWS = 4, SB_LANES = 256;  // block = SB_ROWS rows in flight x SB_LANES beams (coalesced along v)
constexpr int SB_MAX_NV = COSENU_STATIC_MAX_NV;
constexpr int SB_MAX_DEVICES = 64;

// THE scratch: partial[b][4][nv] for the nv of the call in flight, b < SB_BLOCKS.  148 * 4 * 512 doubles = 2 424 832 bytes
// (2.3 MiB) of device memory on every GPU on which this library's device code gets loaded, held until the process exits.
// In HOST code this name is only a stand-in for the symbol (it is not a device address and must never be handed to a
// kernel): host code goes through scratch_of_current_device() below.
static __device__ __align__(256) double g_beam_partials[(size_t)SB_BLOCKS * 4 * SB_MAX_NV];

__device__ __forceinline__ double polarisation_length(double ee, double xx, double re, double im) {
  const double d = ee - xx;
  return sqrt(fma(d, d, 4.0 * fma(re, re, im * im)));   // |P| of rho = (P0 + P.sigma)/2, Eq. (4), un-normalised
}

// pass 1: block b sums its z-range [z0, z1) for every beam: part[b][m][j], m = |P_nu|, P0_nu, |P_nubar|, P0_nubar.
// Same walk as diag_ref_kernel (two rows per thread and trip, row groups added in a fixed order), on the canonical dense
// layout state[8][nz][nv].  Every entry part[b][0..3][0..nv) of every block is written (blocks whose z-range is empty
// write zeros), so nothing in the scratch has to be cleared beforehand and nothing left by an earlier call is ever read.
__global__ void __launch_bounds__(SB_ROWS * SB_LANES)
    beam_partials_kernel(const double* __restrict__ state, double* __restrict__ part, long long nz, int nv) {
  __shared__ double red[SB_ROWS][4][SB_LANES];
  const int tj = threadIdx.x % SB_LANES, tr = threadIdx.x / SB_LANES;
  const long long comp_stride = nz * nv;
  const long long rows_per = (nz + gridDim.x - 1) / gridDim.x;
  const long long z0 = min(nz, blockIdx.x * rows_per), z1 = min(nz, z0 + rows_per);
  for (int j0 = 0; j0 < nv; j0 += SB_LANES) {
    const int j = j0 + tj;
    double a[4] = {0, 0, 0, 0}, b[4] = {0, 0, 0, 0};
    if (j < nv) {
      auto row = [&](long long iz, double (&acc)[4]) {
        const double* q = state + iz * nv + j;
        double c[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) c[k] = q[k * comp_stride];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
          acc[2 * s] += polarisation_length(c[4 * s], c[4 * s + 1], c[4 * s + 2], c[4 * s + 3]);
          acc[2 * s + 1] += c[4 * s] + c[4 * s + 1];
        }
      };
      long long iz = z0 + tr;
      for (; iz + SB_ROWS < z1; iz += 2 * SB_ROWS) { row(iz, a); row(iz + SB_ROWS, b); }
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
        for (int r = 1; r < SB_ROWS; ++r) sum += red[r][m][tj];
        part[((long long)blockIdx.x * 4 + m) * nv + j] = sum;
      }
    }
    __syncthreads();
  }
}

// pass 2: out[m][j] = sum over the SB_BLOCKS partials, in block order, carrying the rounding error of every addition
// along (two-sum), so that the result is the correctly rounded sum of the partials in all but pathological cases -- the
// handle-based path adds the same partials on the host in long double.
__global__ void beam_sums_finish_kernel(const double* __restrict__ part, double* __restrict__ out, int nv, int nblocks) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;   // = m * nv + j
  if (q >= 4 * nv) return;
  double s = 0.0, comp = 0.0;
  for (int b = 0; b < nblocks; ++b) {
    const double x = part[(long long)b * 4 * nv + q];
    const double t = __dadd_rn(s, x);
    const double bb = __dadd_rn(t, -s);
    comp = __dadd_rn(comp, __dadd_rn(__dadd_rn(s, -__dadd_rn(t, -bb)), __dadd_rn(x, -bb)));
    s = t;
  }
  out[q] = __dadd_rn(s, comp);
}

thread_local std::string t_err;   // text of this thread's last failed call

int fail(int code, const std::string& msg) { t_err = "cosenu_beam_sums_static: " + msg; return code; }
int cuda_fail(cudaError_t e, const char* what) {
  (void)cudaGetLastError();   // do not leave the error behind for the caller's next CUDA call
  return fail(COSENU_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// Set-up, once per device and with that device current: ask the runtime where THIS device's copy of g_beam_partials
// lives.  (Every device has its own copy at its own address; the host-side name is none of them.)
std::mutex g_setup_mutex;
double* g_scratch_addr[SB_MAX_DEVICES] = {};

int scratch_of_current_device(int device, double** out) {
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_addr[device]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_beam_partials);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(scratch array)");
    if (!p) return fail(COSENU_ECUDA, "cudaGetSymbolAddress returned a null address for the scratch array");
    g_scratch_addr[device] = static_cast<double*>(p);
  }
  *out = g_scratch_addr[device];
  return COSENU_OK;
}

// a buffer the kernels of `device` can read and write: device memory of that device, or managed memory
int check_device_buffer(const void* p, int device, const char* name) {
  if (!p) return fail(COSENU_EINVAL, std::string(name) + " is NULL");
  if (reinterpret_cast<uintptr_t>(p) % alignof(double)) return fail(COSENU_EINVAL, std::string(name) + " is not aligned for double");
  cudaPointerAttributes at;
  cudaError_t e = cudaPointerGetAttributes(&at, p);
  if (e != cudaSuccess) return cuda_fail(e, "cudaPointerGetAttributes");
  if (at.type == cudaMemoryTypeManaged) return COSENU_OK;
  if (at.type != cudaMemoryTypeDevice)
    return fail(COSENU_EINVAL, std::string(name) + " is a host pointer; this call takes device buffers only");
  if (at.device != device)
    return fail(COSENU_EINVAL, std::string(name) + " belongs to CUDA device " + std::to_string(at.device) + ", but device " +
                                   std::to_string(device) + " is current");
  return COSENU_OK;
}

}  // namespace

extern "C" int cosenu_beam_sums_static(const double* dev_state, int64_t nz, int32_t nv, double* dev_out, void* cuda_stream) {
  if (nv < 1 || nv > SB_MAX_NV)
    return fail(COSENU_EINVAL, "nv = " + std::to_string(nv) + " is outside 1.." + std::to_string(SB_MAX_NV) +
                                   " (COSENU_STATIC_MAX_NV: the built-in scratch array holds 148 x 4 x " +
                                   std::to_string(SB_MAX_NV) + " partial sums); use the handle-based diagnostics for wider v-grids");
  if (nz < 1 || nz > ((int64_t)1 << 40)) return fail(COSENU_EINVAL, "nz = " + std::to_string(nz) + " is outside 1..2^40");
  int device = -1;
  cudaError_t e = cudaGetDevice(&device);
  if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice (no usable CUDA device; there is no CPU fallback)");
  if (device < 0 || device >= SB_MAX_DEVICES) return fail(COSENU_EINVAL, "device ordinal " + std::to_string(device) + " not supported");
  int rc;
  if ((rc = check_device_buffer(dev_state, device, "dev_state"))) return rc;
  if ((rc = check_device_buffer(dev_out, device, "dev_out"))) return rc;
  double* scratch = nullptr;
  if ((rc = scratch_of_current_device(device, &scratch))) return rc;

  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  beam_partials_kernel<<<SB_BLOCKS, SB_ROWS * SB_LANES, 0, stream>>>(dev_state, scratch, (long long)nz, (int)nv);
  if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(e, "launch of beam_partials_kernel");
  const int threads = 256, blocks = (4 * nv + threads - 1) / threads;
  beam_sums_finish_kernel<<<blocks, threads, 0, stream>>>(scratch, dev_out, (int)nv, SB_BLOCKS);
  if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(e, "launch of beam_sums_finish_kernel");
  return COSENU_OK;
}

extern "C" const char* cosenu_beam_sums_static_error(void) { return t_err.c_str(); }
