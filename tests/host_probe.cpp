// host_probe.cpp -- host-side build of the product's stencil arithmetic (weno7_math.h) so that the CPU
// tests can check the formulas the kernels use against the oracle without a GPU.  Test code: built by tests/build_probe.py,
// not by the product's build.
#include "../paper_2203_12866_b200/csrc/weno7_math.h"

extern "C" double cosenu_probe_weno7_face(const double* w7, double v, double eps) {
  // value of f = v u at the interface, as the kernels form it
  return v * cosenu_math::weno7_face(w7, cosenu_math::weno7_beam(v, eps));
}

// two adjacent interfaces from 8 cells (shared differences): out[0] = w[3]|w[4], out[1] = w[4]|w[5]
extern "C" void cosenu_probe_weno7_face2(const double* w8, double v, double eps, double* out) {
  double a, b;
  cosenu_math::weno7_face2(w8, cosenu_math::weno7_beam(v, eps), a, b);
  out[0] = v * a; out[1] = v * b;
}

extern "C" double cosenu_probe_fd4_ko3(const double* u5, double v, double dz, double eps_ko) {
  return cosenu_math::fd4_ko3(u5[0], u5[1], u5[2], u5[3], u5[4], -v / (12.0 * dz), -eps_ko / (16.0 * dz));
}

extern "C" double cosenu_probe_fd4_ko5(const double* u7, double v, double dz, double eps_ko) {
  return cosenu_math::fd4_ko5(u7[0], u7[1], u7[2], u7[3], u7[4], u7[5], u7[6], -v / (12.0 * dz), eps_ko / (64.0 * dz));
}
