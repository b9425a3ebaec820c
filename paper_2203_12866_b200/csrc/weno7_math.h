// weno7_math.h -- per-interface arithmetic of the product's WENO7 and FD4+KO3 stencils.
//
// Compiles as CUDA device code (stage_kernels.cuh) and as plain host C++ (host_probe.cpp, used only by
// the CPU tests to check these formulas without a GPU).  Shares nothing with oracle/.
//
// WENO7 (App. A / Algorithm 1; Eqs. (12)-(14) PAPER.md:134-145).
// The paper prints the smoothness indicators SI_r as 10-term polynomials in the four cell values of
// sub-stencil S_r (Eq. A.3).  They vanish on constants, so they are quadratic forms in the three
// undivided first differences x, y, z of S_r.  Writing the cubic p_r(xi) = a0 + a1 xi + a2 xi^2 + a3 xi^3
// that has the four cell averages of S_r (xi in cell widths, centred on cell i), the printed SI_r are
// exactly 240 * sum_{l=1..3} int_{-1/2}^{1/2} (d^l p_r / d xi^l)^2 d xi, which diagonalises to
//      SI_r = 240 A_r^2 + 260 s_r^2 + (781/3) t_r^2,
//      A_r = a1 + a3/4,   s_r = 2 a2,   t_r = 6 a3 (the third difference of S_r),
// and the 4th-order candidate of Eq. (A.2) is   fhat_r = u_i + A_r/2 + s_r/12.
// (Derived for this file from the printed coefficients; the derivation is restated in DESIGN.md.)
// With p = y - x, q = z - y (second differences), t = q - p:
//      r=0 (S_0 = i..i+3):   A = x - (5/6)p + (1/3)q,   s = p - t
//      r=1 (S_1 = i-1..i+2): A = x + (2/3)p - (1/6)q,   s = p
//      r=2 (S_2 = i-2..i+1): A = x + (7/6)p + (1/3)q,   s = q
//      r=3 (S_3 = i-3..i):   A = x + (2/3)p + (11/6)q,  s = q + t
// The difference form needs ~80 fp64 instructions per interface instead of ~140 and has no
// catastrophic cancellation for nearly constant data.
//
// Linear weights (PAPER.md:372 prints them in the reverse order of its own r labels; only
// d_0..d_3 = 4/35, 18/35, 12/35, 1/35 reproduces Eq. (A.1), reading A6).
//
// The reconstruction acts on f = v u with v constant along z (reading A8), so
// SI_r[f] = v^2 SI_r[u] and  fhat[f] = v fhat[u]:  the routines work on u.
// The nonlinear weights  w_r = d_r / (SI_r + eps)^2  (Eq. 14) are combined with ONE division.  With
//      qs_r = (SI_r[u] + eps/v^2) / sqrt(d_r)        (so that  w_r  is proportional to  1 / qs_r^2),
//      P_r  = prod_{m != r} qs_m^2,
//      F = sum_r w_r fhat_r / sum_r w_r = u_i + (1/2) [sum_r P_r (A_r + s_r/6)] / [sum_r P_r].
// The per-beam constants  eps_r = (eps/v^2)/sqrt(d_r)  are formed once per beam (Weno7Beam).
// Range: needs |u|^2 * 1e4 / v^2-scaled terms to stay below ~1e50 per factor (states are O(1)); eps / v^2 is
// clamped to <= 1e45 (the flux is multiplied by v afterwards, so v = 0 gives exactly 0); 1e-40 <= eps <= 1e30.
#ifndef COSENU_WENO7_MATH_H
#define COSENU_WENO7_MATH_H

#ifdef __CUDACC__
#define COSENU_HD __host__ __device__ __forceinline__
#else
#include <cmath>
#define COSENU_HD inline
using std::fma;
#endif

namespace cosenu_math {

// 1/(2d): hardware seed (MUFU.RCP64H) + one third-order step (3 FMA instead of the 4 of two Newton steps; relative error
// <= |e|^3 ~ 2^-57 + rounding) on the device, plain division on the host.  The factor 1/2
// of "F = u_i + (1/2) num/den" costs no fp64 instruction: 2d is an exponent increment (integer add on the high word), and
// every quantity of the iteration is then an exact power-of-two multiple of the plain reciprocal's.  d > 0, finite, normal.
COSENU_HD double fast_half_rcp(double d) {
#ifdef __CUDA_ARCH__
  const double d2 = __hiloint2double(__double2hiint(d) + 0x00100000, __double2loint(d));
  double x;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d2));
  const double e = fma(-d2, x, 1.0);   // |e| <= 2^-19: the seed sees the upper 32 bits of d2
  const double t = fma(e, e, e);       // 1/(1 - e) = 1 + e + e^2 + O(e^3)
  return fma(x, t, x);
#else
  return 0.5 / d;
#endif
}

// per-beam constants of the weights: eps_r = (eps / v^2) / sqrt(d_r), d = (4, 18, 12, 1)/35
struct Weno7Beam {
  double e0, e1, e2, e3;
};
// Host and device builds of this routine are NOT bit-identical: the device forms eps / v^2 from the reciprocal seed plus
// one third-order step (about 1 ulp), the host divides, so e_r may differ by an ulp or two between them; the host-probe pins
// (tests/host_probe.cpp) check the formula, tests/device_probe.cu + test_gpu_parity.py::test_device_beam_constants check the
// device's numbers against eps / v^2 over the accepted range of eps.  Clamping: v^2 below 1e-300 counts as 1e-300 and
// eps / v^2 above 1e45 as 1e45.  The oracle clamps nothing; the two differ only where (SI + eps/v^2) is eps/v^2 to working
// precision anyway (weights = d_r, the linear scheme) and the flux carries the factor |v| <= 1e-8.
COSENU_HD Weno7Beam weno7_beam(double v, double eps) {
  // eps / v^2, kept below 1e45 so that the products of six q_r stay in range for every accepted eps (1e-40 .. 1e30), also
  // on a beam with v = 0 exactly (vertex-centred grids); there the flux is multiplied by |v| = 0 afterwards
  const double v2 = v * v;
  const double v2c = v2 < 1e-300 ? 1e-300 : v2;
#ifdef __CUDA_ARCH__
  // eps / v^2 once per beam and work item: the hardware seed + one third-order step (as in fast_half_rcp; ~1 ulp) instead of
  // the ~40 dependent instructions of an IEEE division, which the marching warps would run serially at every item
  double x;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(v2c));
  const double e = fma(-v2c, x, 1.0);
  double ev = eps * fma(x, fma(e, e, e), x);
#else
  double ev = eps / v2c;
#endif
  if (ev > 1e45) ev = 1e45;
  Weno7Beam b;
  b.e0 = ev * 2.9580398915498080213;   // sqrt(35/4)
  b.e1 = ev * 1.3944333775567926;      // sqrt(35/18)
  b.e2 = ev * 1.7078251276599330;      // sqrt(35/12)
  b.e3 = ev * 5.9160797830996160426;   // sqrt(35)
  return b;
}

// the 19 constants of weno7_core.  On the device they live in the constant bank, so that every DFMA takes its constant as an
// operand (c[bank][offset]); as 64-bit immediates they would be re-materialised into uniform registers (two UMOV each) at
// every work item.  k_r = 1/sqrt(d_r) = sqrt(35/4), sqrt(35/18), sqrt(35/12), sqrt(35).
enum { C_1_3, C_M5_6, C_M1_6, C_2_3, C_7_6, C_11_6, C_1_6, C_240K0, C_260K0, C_781K0, C_240K1, C_260K1, C_781K1,
       C_240K2, C_260K2, C_781K2, C_240K3, C_260K3, C_781K3, C_COUNT };
#define COSENU_WENO_CONSTANTS                                                                                              \
  {1.0 / 3.0, -5.0 / 6.0, -1.0 / 6.0, 2.0 / 3.0, 7.0 / 6.0, 11.0 / 6.0, 1.0 / 6.0,                                          \
   240.0 * 2.9580398915498080213, 260.0 * 2.9580398915498080213, (781.0 / 3.0) * 2.9580398915498080213,                   \
   240.0 * 1.3944333775567926, 260.0 * 1.3944333775567926, (781.0 / 3.0) * 1.3944333775567926,                            \
   240.0 * 1.7078251276599330, 260.0 * 1.7078251276599330, (781.0 / 3.0) * 1.7078251276599330,                            \
   240.0 * 5.9160797830996160426, 260.0 * 5.9160797830996160426, (781.0 / 3.0) * 5.9160797830996160426}
#ifdef __CUDACC__
__constant__ double weno_const_dev[C_COUNT] = COSENU_WENO_CONSTANTS;
#endif
static constexpr double weno_const_host[C_COUNT] = COSENU_WENO_CONSTANTS;
#ifdef __CUDA_ARCH__
#define WC(i) weno_const_dev[i]
#else
#define WC(i) weno_const_host[i]
#endif

// the part of Algorithm 1 after the undivided differences: D[0..5], E[0..4], T[0..3] of the 7 cells
// w[0..6] (D_k = w[k+1]-w[k], E_k = D[k+1]-D[k], T_k = E[k+1]-E[k]); ui = w[3]; TTk = T_k^2 (shared
// between neighbouring interfaces by weno7_face2).
COSENU_HD double weno7_core(double ui, double D0, double D1, double D2, double D3, double E0, double E1, double E2,
                            double E3, double E4, double T0, double T3, double TT0, double TT1, double TT2, double TT3,
                            const Weno7Beam& bm) {
  // A_r, s_r per sub-stencil: (x, p, q, t) = (D[3-r], E[3-r], E[4-r], T[3-r])
  const double A0 = fma(WC(C_1_3), E4, fma(WC(C_M5_6), E3, D3));
  const double A1 = fma(WC(C_M1_6), E3, fma(WC(C_2_3), E2, D2));
  const double A2 = fma(WC(C_1_3), E2, fma(WC(C_7_6), E1, D1));
  const double A3 = fma(WC(C_11_6), E1, fma(WC(C_2_3), E0, D0));
  const double s0 = E3 - T3, s3 = E1 + T0;   // s1 = s2 = E2
  const double ss12 = E2 * E2;
  // qs_r = (240 A^2 + 260 s^2 + (781/3) t^2 + eps/v^2) / sqrt(d_r)
  const double q0 = fma(WC(C_240K0), A0 * A0, fma(WC(C_260K0), s0 * s0, fma(WC(C_781K0), TT3, bm.e0)));
  const double q1 = fma(WC(C_240K1), A1 * A1, fma(WC(C_260K1), ss12, fma(WC(C_781K1), TT2, bm.e1)));
  const double q2 = fma(WC(C_240K2), A2 * A2, fma(WC(C_260K2), ss12, fma(WC(C_781K2), TT1, bm.e2)));
  const double q3 = fma(WC(C_240K3), A3 * A3, fma(WC(C_260K3), s3 * s3, fma(WC(C_781K3), TT0, bm.e3)));
  const double Q0 = q0 * q0, Q1 = q1 * q1, Q2 = q2 * q2, Q3 = q3 * q3;
  const double Q01 = Q0 * Q1, Q23 = Q2 * Q3;
  // P_0 = Q1 Q23, P_1 = Q0 Q23, P_2 = Q01 Q3, P_3 = Q01 Q2, grouped:
  //   den = Q23 (Q0 + Q1) + Q01 (Q2 + Q3),  num = Q23 (Q1 c0 + Q0 c1) + Q01 (Q3 c2 + Q2 c3)
  const double c0 = fma(WC(C_1_6), s0, A0), c1 = fma(WC(C_1_6), E2, A1), c2 = fma(WC(C_1_6), E2, A2),
               c3 = fma(WC(C_1_6), s3, A3);
  const double den = fma(Q01, Q2 + Q3, Q23 * (Q0 + Q1));
  const double num = fma(Q01, fma(Q3, c2, Q2 * c3), Q23 * fma(Q1, c0, Q0 * c1));
  return fma(num, fast_half_rcp(den), ui);
}

// WENO7 value of u at the interface between w[3] and w[4], biased towards w[0] (the upwind side):
// w[0..6] = u_{i-3} .. u_{i+3} for v >= 0; the mirrored cells u_{i+4} .. u_{i-2} for v < 0.
COSENU_HD double weno7_face(const double w[7], const Weno7Beam& bm) {
  const double D0 = w[1] - w[0], D1 = w[2] - w[1], D2 = w[3] - w[2], D3 = w[4] - w[3], D4 = w[5] - w[4],
               D5 = w[6] - w[5];
  const double E0 = D1 - D0, E1 = D2 - D1, E2 = D3 - D2, E3 = D4 - D3, E4 = D5 - D4;
  const double T0 = E1 - E0, T1 = E2 - E1, T2 = E3 - E2, T3 = E4 - E3;
  return weno7_core(w[3], D0, D1, D2, D3, E0, E1, E2, E3, E4, T0, T3, T0 * T0, T1 * T1, T2 * T2, T3 * T3, bm);
}

// two adjacent interfaces from 8 cells w[0..7] with shared differences:
//   Fa = interface between w[3] and w[4],  Fb = interface between w[4] and w[5], both biased towards w[0].
COSENU_HD void weno7_face2(const double w[8], const Weno7Beam& bm, double& Fa, double& Fb) {
  const double D0 = w[1] - w[0], D1 = w[2] - w[1], D2 = w[3] - w[2], D3 = w[4] - w[3], D4 = w[5] - w[4],
               D5 = w[6] - w[5], D6 = w[7] - w[6];
  const double E0 = D1 - D0, E1 = D2 - D1, E2 = D3 - D2, E3 = D4 - D3, E4 = D5 - D4, E5 = D6 - D5;
  const double T0 = E1 - E0, T1 = E2 - E1, T2 = E3 - E2, T3 = E4 - E3, T4 = E5 - E4;
  const double TT0 = T0 * T0, TT1 = T1 * T1, TT2 = T2 * T2, TT3 = T3 * T3, TT4 = T4 * T4;
  Fa = weno7_core(w[3], D0, D1, D2, D3, E0, E1, E2, E3, E4, T0, T3, TT0, TT1, TT2, TT3, bm);
  Fb = weno7_core(w[4], D1, D2, D3, D4, E1, E2, E3, E4, E5, T1, T4, TT1, TT2, TT3, TT4, bm);
}

// FD4 + KO3 in difference form (Eq. (5)): returns
//   cadv * (u_{i-2} - 8u_{i-1} + 8u_{i+1} - u_{i+2}) + cko * (u_{i-2} - 4u_{i-1} + 6u_i - 4u_{i+1} + u_{i+2})
// with cadv = -v/(12 dz), cko = -eps_ko/(16 dz) (dissipative sign, reading A4).
// Written on first differences so that z-uniform data gives exactly 0.
COSENU_HD double fd4_ko3(double um2, double um1, double u0, double up1, double up2, double cadv, double cko) {
  const double a = um1 - um2, b = u0 - um1, c = up1 - u0, d = up2 - up1;
  const double central = fma(-7.0, b + c, a + d);        // = -(u_{i-2} - 8u_{i-1} + 8u_{i+1} - u_{i+2})
  const double fourth = fma(-3.0, c - b, d - a);         // = u_{i+2} - 4u_{i+1} + 6u_i - 4u_{i-1} + u_{i-2}
  return fma(-cadv, central, cko * fourth);
}

// FD4 + Kreiss-Oliger of order r = 3 (Eq. (5) PAPER.md:88-92 with r = 3: a 7-point operator): returns
//   cadv * (u_{i-2} - 8u_{i-1} + 8u_{i+1} - u_{i+2}) + cko6 * (u_{i-3} - 6u_{i-2} + 15u_{i-1} - 20u_i + 15u_{i+1} - 6u_{i+2} + u_{i+3})
// with cadv = -v/(12 dz), cko6 = +eps_ko/(64 dz): (D+ D-)^3 has the symbol -64 sin^6(k dz/2)/dz^6, so the dissipative
// sign (reading A4) is PLUS the sixth difference.  On first differences, exactly 0 on z-uniform data.
COSENU_HD double fd4_ko5(double um3, double um2, double um1, double u0, double up1, double up2, double up3, double cadv,
                         double cko6) {
  const double a = um2 - um3, b = um1 - um2, c = u0 - um1, d = up1 - u0, e = up2 - up1, f = up3 - up2;
  const double central = fma(-7.0, c + d, b + e);
  const double sixth = fma(10.0, d - c, fma(-5.0, e - b, f - a));
  return fma(-cadv, central, cko6 * sixth);
}

}  // namespace cosenu_math
#endif
