// device_probe.cu -- DEVICE-side build of the product's per-beam WENO constants (csrc/weno7_math.h) so that a GPU test can look at
// the numbers the kernels really use: on the device eps / v^2 comes from the hardware reciprocal seed plus one correction
// step, on the host (host_probe.cpp) from a division.  Test code: built by tests/build_probe.py, not part of the product.
#include "../paper_2203_12866_b200/csrc/weno7_math.h"

#include <cuda_runtime.h>

__global__ void probe_beam_kernel(const double* __restrict__ v, const double* __restrict__ eps, double* __restrict__ out, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const cosenu_math::Weno7Beam b = cosenu_math::weno7_beam(v[i], eps[i]);
  out[4 * i] = b.e0; out[4 * i + 1] = b.e1; out[4 * i + 2] = b.e2; out[4 * i + 3] = b.e3;
}

// dev_v[n], dev_eps[n] -> dev_out[n][4] = (e0, e1, e2, e3); device pointers, synchronises; returns the cudaError_t
extern "C" int cosenu_device_probe_weno7_beam(const double* dev_v, const double* dev_eps, double* dev_out, int n) {
  probe_beam_kernel<<<(n + 127) / 128, 128>>>(dev_v, dev_eps, dev_out, n);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  return (int)e;
}
