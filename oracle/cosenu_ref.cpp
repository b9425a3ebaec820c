// cosenu_ref.cpp -- CPU ORACLE for the COSEnu RK4 hot path (arXiv 2203.12866).
//
// TEST INFRASTRUCTURE ONLY (see cosenu_ref.h).  Plain loops, fp64, no blocking, no fusion,
// no reordering beyond what the cited passage states.  Moments are summed in long double so
// that the oracle is the more accurate side.  Build: g++ -O2 -ffp-contract=off -fopenmp.
// Shares nothing with paper_2203_12866_b200/csrc/.
//
// Readings of the paper used here are the ones listed in DESIGN.md ("Readings", A1..A16).

#include "cosenu_ref.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#else
static inline int omp_get_max_threads() { return 1; }
#endif

struct cosenu_ref {
  int64_t nz; int32_t nv;
  double L, dt, omega, theta, mu; int scheme;
  double eps_ko = 0.1;      // PAPER.md:164 "KO3 with eps_KO = 0.1"
  double weno_eps = 1e-6;   // PAPER.md:145 "typical value ~1e-6"
  int advect = 1; int threads = 0; int quad = 0;
  int ko_r = 2;             // order r of the Kreiss-Oliger operator, Eq. (5): "we have used r = 2 for most"
  double dz, dv;
  std::vector<double> v;    // beam velocities: bin centres or vertex-centred points
  std::vector<double> wq;   // quadrature weights in units of dv: int f dv ~ dv * sum_j wq_j f(v_j)
  std::vector<double> y;    // current state, canonical layout [8][nz][nv]
  bool have_state = false;
  double t = 0; int64_t step = 0;
  // references taken at t = 0 (set_state / init) for the diagnostics
  double sum_ee0[2] = {0, 0};
  std::vector<double> Pref[2], P0ref[2];
  double M0_init[3] = {0, 0, 0};
  std::string err;
};

static std::string g_err;  // last error of a failed create

static inline int64_t wrap(int64_t i, int64_t n) { return ((i % n) + n) % n; }

// v-grid and quadrature weights (readings A1 and section 3.1 of the paper)
static void build_vgrid(cosenu_ref* h) {
  const int nv = h->nv;
  h->v.resize(nv); h->wq.assign(nv, 1.0);
  if (h->quad == 0) {             // bins [v_j, v_j + dv] represented by their centres; simple Riemann sum
    h->dv = 2.0 / (double)nv;
    for (int j = 0; j < nv; ++j) h->v[j] = -1.0 + (j + 0.5) * h->dv;
  } else {                        // fixed-width vertex-centred points over [-1, 1]
    h->dv = 2.0 / (double)(nv - 1);
    for (int j = 0; j < nv; ++j) h->v[j] = -1.0 + (double)j * h->dv;
    if (h->quad == 1) {           // trapezoid rule
      h->wq[0] = h->wq[nv - 1] = 0.5;
    } else {                      // Simpson's rule: (1, 4, 2, 4, ..., 4, 1)/3
      for (int j = 0; j < nv; ++j) h->wq[j] = (j == 0 || j == nv - 1) ? 1.0 / 3.0 : ((j & 1) ? 4.0 / 3.0 : 2.0 / 3.0);
    }
  }
}
static inline size_t idx(const cosenu_ref* h, int c, int64_t iz, int iv) {
  return ((size_t)c * h->nz + iz) * h->nv + iv;
}

// ---------------------------------------------------------------- App. A
// f[0..6] = f_{i-3} .. f_{i+3};  f[3] is cell i.
extern "C" void cosenu_ref_weno7_candidates(const double f[7], double fh[4]) {
  const double *m3 = f, *m2 = f + 1, *m1 = f + 2, *c = f + 3, *p1 = f + 4, *p2 = f + 5, *p3 = f + 6;
  // Eq. (A.2a-d)
  fh[0] = (3.0 / 12.0) * *c + (13.0 / 12.0) * *p1 + (-5.0 / 12.0) * *p2 + (1.0 / 12.0) * *p3;
  fh[1] = (-1.0 / 12.0) * *m1 + (7.0 / 12.0) * *c + (7.0 / 12.0) * *p1 + (-1.0 / 12.0) * *p2;
  fh[2] = (1.0 / 12.0) * *m2 + (-5.0 / 12.0) * *m1 + (13.0 / 12.0) * *c + (3.0 / 12.0) * *p1;
  fh[3] = (-3.0 / 12.0) * *m3 + (13.0 / 12.0) * *m2 + (-23.0 / 12.0) * *m1 + (25.0 / 12.0) * *c;
}

extern "C" void cosenu_ref_weno7_si(const double f[7], double si[4]) {
  const double m3 = f[0], m2 = f[1], m1 = f[2], c = f[3], p1 = f[4], p2 = f[5], p3 = f[6];
  // Eq. (A.3a-d) exactly as printed
  si[0] = c * (2107 * c - 9402 * p1 + 7042 * p2 - 1854 * p3)
        + p1 * (11003 * p1 - 17246 * p2 + 4642 * p3)
        + p2 * (7043 * p2 - 3882 * p3) + 547 * p3 * p3;
  si[1] = m1 * (547 * m1 - 2522 * c + 1922 * p1 - 494 * p2)
        + c * (3443 * c - 5966 * p1 + 1602 * p2)
        + p1 * (2843 * p1 - 1642 * p2) + 267 * p2 * p2;
  si[2] = m2 * (267 * m2 - 1642 * m1 + 1602 * c - 494 * p1)
        + m1 * (2843 * m1 - 5966 * c + 1922 * p1)
        + c * (3443 * c - 2522 * p1) + 547 * p1 * p1;
  si[3] = m3 * (547 * m3 - 3882 * m2 + 4642 * m1 - 1854 * c)
        + m2 * (7043 * m2 - 17246 * m1 + 7042 * c)
        + m1 * (11003 * m1 - 9402 * c) + 2107 * c * c;
}

extern "C" void cosenu_ref_weno7_dr(double d[4]) {
  // PAPER.md:372 prints 1/35, 12/35, 18/35, 4/35 for d0..d3; with the paper's own S_r labels
  // only the reversed order reproduces Eq. (A.1) (reading A6).
  d[0] = 4.0 / 35.0; d[1] = 18.0 / 35.0; d[2] = 12.0 / 35.0; d[3] = 1.0 / 35.0;
}

extern "C" double cosenu_ref_weno7_face(const double f[7], double eps) {
  // Algorithm 1; Eqs. (13), (14) PAPER.md:139-143
  double fh[4], si[4], d[4], w[4];
  cosenu_ref_weno7_candidates(f, fh);
  cosenu_ref_weno7_si(f, si);
  cosenu_ref_weno7_dr(d);
  double wsum = 0;
  for (int r = 0; r < 4; ++r) { w[r] = d[r] / ((si[r] + eps) * (si[r] + eps)); wsum += w[r]; }
  double F = 0;
  for (int r = 0; r < 4; ++r) F += (w[r] / wsum) * fh[r];
  return F;
}

// ---------------------------------------------------------------- moments (S1)
// M^k_X(z) = dv * sum_j v_j^k X(z,j), X = D = rho - rho_bar^* (Eq. 3a), Riemann sum PAPER.md:78
static void moments(const cosenu_ref* h, const double* y, double* M /*[6][nz]*/) {
  const int64_t nz = h->nz; const int nv = h->nv;
#pragma omp parallel for schedule(static) num_threads(h->threads > 0 ? h->threads : omp_get_max_threads())
  for (int64_t i = 0; i < nz; ++i) {
    long double s[6] = {0, 0, 0, 0, 0, 0};
    for (int j = 0; j < nv; ++j) {
      double Dd = (y[idx(h, 0, i, j)] - y[idx(h, 1, i, j)]) - (y[idx(h, 4, i, j)] - y[idx(h, 5, i, j)]);
      double Dr = y[idx(h, 2, i, j)] - y[idx(h, 6, i, j)];
      double Di = y[idx(h, 3, i, j)] + y[idx(h, 7, i, j)];  // conj of rho_bar flips Im only
      const long double vj = h->v[j], w = h->wq[j];
      s[0] += w * Dd; s[1] += w * (vj * Dd); s[2] += w * Dr; s[3] += w * (vj * Dr); s[4] += w * Di; s[5] += w * (vj * Di);
    }
    for (int m = 0; m < 6; ++m) M[(size_t)m * nz + i] = (double)(s[m] * (long double)h->dv);
  }
}

// ---------------------------------------------------------------- RHS = advection + commutator
static void rhs(const cosenu_ref* h, const double* y, double* k) {
  const int64_t nz = h->nz; const int nv = h->nv;
  const int nthreads = h->threads > 0 ? h->threads : omp_get_max_threads();
  std::vector<double> M((size_t)6 * nz);
  moments(h, y, M.data());

  // --- advection term, component by component (PAPER.md:82-92 / 98-145)
  if (!h->advect) {
    std::memset(k, 0, sizeof(double) * 8 * (size_t)nz * nv);
  } else if (h->scheme == COSENU_REF_FD4_KO3) {
#pragma omp parallel for schedule(static) num_threads(nthreads)
    for (int64_t i = 0; i < nz; ++i) {
      const int64_t im2 = wrap(i - 2, nz), im1 = wrap(i - 1, nz), ip1 = wrap(i + 1, nz), ip2 = wrap(i + 2, nz);
      for (int c = 0; c < 8; ++c)
        for (int j = 0; j < nv; ++j) {
          const double um2 = y[idx(h, c, im2, j)], um1 = y[idx(h, c, im1, j)], u0 = y[idx(h, c, i, j)],
                       up1 = y[idx(h, c, ip1, j)], up2 = y[idx(h, c, ip2, j)];
          // 4th-order central difference
          const double dudz = (um2 - 8.0 * um1 + 8.0 * up1 - up2) / (12.0 * h->dz);
          // Kreiss-Oliger r=2, Eq. (5) with the dissipative sign (reading A4):
          //   Q u = -(eps/16 dz) (u_{i-2} - 4u_{i-1} + 6u_i - 4u_{i+1} + u_{i+2})
          double ko = (h->eps_ko / (16.0 * h->dz)) * (um2 - 4.0 * um1 + 6.0 * u0 - 4.0 * up1 + up2);
          if (h->ko_r == 3) {
            // Eq. (5) with r = 3: eps h^5 (D+ D-)^3 / 2^6 = (eps / 64 dz) (u_{i-3} - 6u_{i-2} + 15u_{i-1} - 20u_i + 15u_{i+1}
            // - 6u_{i+2} + u_{i+3}); dissipative sign (reading A4): its Fourier symbol is -(eps/dz) sin^6(k dz/2), so it is
            // ADDED here where the r = 2 term is subtracted ((D+ D-)^r alternates in sign with r)
            const double um3 = y[idx(h, c, wrap(i - 3, nz), j)], up3 = y[idx(h, c, wrap(i + 3, nz), j)];
            ko = -(h->eps_ko / (64.0 * h->dz)) * (um3 - 6.0 * um2 + 15.0 * um1 - 20.0 * u0 + 15.0 * up1 - 6.0 * up2 + up3);
          }
          k[idx(h, c, i, j)] = -h->v[j] * dudz - ko;
        }
    }
  } else {
    // finite volume, Eq. (7): d u_i/dt = -(F_{i+1/2} - F_{i-1/2})/dz, F from Algorithm 1 on f = v u
    // (reading A8), upwinded by the sign of v (reading A9).  One flux per interface.
    std::vector<double> F((size_t)nz * nv);
    for (int c = 0; c < 8; ++c) {
#pragma omp parallel for schedule(static) num_threads(nthreads)
      for (int64_t i = 0; i < nz; ++i)
        for (int j = 0; j < nv; ++j) {
          const double vj = h->v[j];
          double f[7];
          if (vj >= 0) {
            for (int m = -3; m <= 3; ++m) f[m + 3] = vj * y[idx(h, c, wrap(i + m, nz), j)];
          } else {
            // mirror image about the interface i+1/2: g_m = f_{(2i+1)-m}
            for (int m = -3; m <= 3; ++m) f[m + 3] = vj * y[idx(h, c, wrap(i + 1 - m, nz), j)];
          }
          F[(size_t)i * nv + j] = cosenu_ref_weno7_face(f, h->weno_eps);
        }
#pragma omp parallel for schedule(static) num_threads(nthreads)
      for (int64_t i = 0; i < nz; ++i) {
        const int64_t im1 = wrap(i - 1, nz);
        for (int j = 0; j < nv; ++j)
          k[idx(h, c, i, j)] = -(F[(size_t)i * nv + j] - F[(size_t)im1 * nv + j]) / h->dz;
      }
    }
  }

  // --- commutator -i[H,rho], -i[Hbar,rho_bar] (Eq. 1, 3)
  const double c2t = std::cos(2.0 * h->theta), s2t = std::sin(2.0 * h->theta);
#pragma omp parallel for schedule(static) num_threads(nthreads)
  for (int64_t i = 0; i < nz; ++i) {
    const double M0d = M[0 * (size_t)nz + i], M1d = M[1 * (size_t)nz + i];
    const double M0r = M[2 * (size_t)nz + i], M1r = M[3 * (size_t)nz + i];
    const double M0i = M[4 * (size_t)nz + i], M1i = M[5 * (size_t)nz + i];
    for (int j = 0; j < nv; ++j) {
      const double vj = h->v[j];
      // mu * int dv' (1 - v v') D(v') = mu (M^0 - v M^1)
      const double Sd = h->mu * (M0d - vj * M1d), Sr = h->mu * (M0r - vj * M1r), Si = h->mu * (M0i - vj * M1i);
      for (int s = 0; s < 2; ++s) {
        // H (s=0): H_vac + S ;  Hbar (s=1): H_vac - S^*   (Eq. 3a / 3b)
        const double A  = -h->omega * c2t + (s == 0 ? Sd : -Sd);          // H_ee - H_xx
        const double Br = 0.5 * h->omega * s2t + (s == 0 ? Sr : -Sr);     // Re H_ex
        const double Bi = (s == 0 ? Si : Si);                             // Im H_ex ; -(S^*) keeps +Si
        const int o = 4 * s;
        const double ee = y[idx(h, o + 0, i, j)], xx = y[idx(h, o + 1, i, j)];
        const double r = y[idx(h, o + 2, i, j)], im = y[idx(h, o + 3, i, j)];
        const double T = 2.0 * (Bi * r - Br * im);
        k[idx(h, o + 0, i, j)] += T;
        k[idx(h, o + 1, i, j)] -= T;
        k[idx(h, o + 2, i, j)] += A * im - Bi * (ee - xx);
        k[idx(h, o + 3, i, j)] += -A * r + Br * (ee - xx);
      }
    }
  }
}

// ---------------------------------------------------------------- classical RK4
static void rk4_step(cosenu_ref* h) {
  const size_t n = 8 * (size_t)h->nz * h->nv;
  std::vector<double> k1(n), k2(n), k3(n), k4(n), ys(n);
  const double dt = h->dt;
  rhs(h, h->y.data(), k1.data());
  for (size_t q = 0; q < n; ++q) ys[q] = h->y[q] + 0.5 * dt * k1[q];
  rhs(h, ys.data(), k2.data());
  for (size_t q = 0; q < n; ++q) ys[q] = h->y[q] + 0.5 * dt * k2[q];
  rhs(h, ys.data(), k3.data());
  for (size_t q = 0; q < n; ++q) ys[q] = h->y[q] + dt * k3[q];
  rhs(h, ys.data(), k4.data());
  for (size_t q = 0; q < n; ++q) h->y[q] = h->y[q] + (dt / 6.0) * (k1[q] + 2.0 * k2[q] + 2.0 * k3[q] + k4[q]);
  h->t += dt; h->step += 1;
}

// ---------------------------------------------------------------- diagnostics
static double plen(const double* y, const cosenu_ref* h, int s, int64_t i, int j) {
  const int o = 4 * s;
  const double d = y[idx(h, o, i, j)] - y[idx(h, o + 1, i, j)];
  const double r = y[idx(h, o + 2, i, j)], im = y[idx(h, o + 3, i, j)];
  return std::sqrt(d * d + 4.0 * (r * r + im * im));  // |P| of Eq. (4), un-normalised
}

static void m0_vector(const cosenu_ref* h, const double* y, double M0[3]) {
  long double s[3] = {0, 0, 0};
  for (int64_t i = 0; i < h->nz; ++i)
    for (int j = 0; j < h->nv; ++j) {
      const double Dd = (y[idx(h, 0, i, j)] - y[idx(h, 1, i, j)]) - (y[idx(h, 4, i, j)] - y[idx(h, 5, i, j)]);
      const double Dr = y[idx(h, 2, i, j)] - y[idx(h, 6, i, j)];
      const double Di = y[idx(h, 3, i, j)] + y[idx(h, 7, i, j)];
      const long double w = h->wq[j];
      s[0] += w * (2.0 * Dr); s[1] += w * (-2.0 * Di); s[2] += w * Dd;  // P = (2 Re, -2 Im, ee - xx)
    }
  for (int m = 0; m < 3; ++m) M0[m] = (double)(s[m] * (long double)(h->dz * h->dv));
}

static void take_references(cosenu_ref* h) {
  for (int s = 0; s < 2; ++s) {
    h->Pref[s].assign(h->nv, 0.0); h->P0ref[s].assign(h->nv, 0.0);
    long double see = 0;
    for (int j = 0; j < h->nv; ++j) {
      long double sp = 0, s0 = 0;
      for (int64_t i = 0; i < h->nz; ++i) {
        sp += plen(h->y.data(), h, s, i, j);
        s0 += h->y[idx(h, 4 * s, i, j)] + h->y[idx(h, 4 * s + 1, i, j)];
        see += (long double)h->wq[j] * h->y[idx(h, 4 * s, i, j)];
      }
      h->Pref[s][j] = (double)(sp / h->nz); h->P0ref[s][j] = (double)(s0 / h->nz);
    }
    h->sum_ee0[s] = (double)see;
  }
  m0_vector(h, h->y.data(), h->M0_init);
}

// ================================================================ C ABI
extern "C" cosenu_ref_t* cosenu_ref_create(int64_t nz, int32_t nv, double L, double dt, double omega,
                                           double theta, double mu, int scheme) {
  if (nz < 16 || nv < 2 || !(L > 0) || !(dt > 0) || (scheme != 0 && scheme != 1) ||
      !std::isfinite(omega) || !std::isfinite(theta) || !std::isfinite(mu)) {
    g_err = "cosenu_ref_create: invalid argument"; return nullptr;
  }
  cosenu_ref* h = new (std::nothrow) cosenu_ref();
  if (!h) { g_err = "out of memory"; return nullptr; }
  h->nz = nz; h->nv = nv; h->L = L; h->dt = dt; h->omega = omega; h->theta = theta; h->mu = mu; h->scheme = scheme;
  h->dz = L / (double)nz;
  build_vgrid(h);
  try { h->y.assign(8 * (size_t)nz * nv, 0.0); } catch (...) { delete h; g_err = "out of memory"; return nullptr; }
  return h;
}

extern "C" int cosenu_ref_set_option(cosenu_ref_t* h, int key, double value) {
  if (!h) return COSENU_REF_EINVAL;
  switch (key) {
    case COSENU_REF_OPT_EPS_KO: if (!(value >= 0)) break; h->eps_ko = value; return COSENU_REF_OK;
    case COSENU_REF_OPT_WENO_EPS: if (!(value > 0)) break; h->weno_eps = value; return COSENU_REF_OK;
    case COSENU_REF_OPT_ADVECT: h->advect = value != 0; return COSENU_REF_OK;
    case COSENU_REF_OPT_THREADS: if (value < 0) break; h->threads = (int)value; return COSENU_REF_OK;
    case COSENU_REF_OPT_KO_ORDER: if (value != 2 && value != 3) break; h->ko_r = (int)value; return COSENU_REF_OK;
    case COSENU_REF_OPT_QUADRATURE:
      if ((value != 0 && value != 1 && value != 2) || h->have_state || (value == 2 && (h->nv % 2 == 0 || h->nv < 3))) break;
      h->quad = (int)value; build_vgrid(h); return COSENU_REF_OK;
  }
  h->err = "cosenu_ref_set_option: bad key or value"; return COSENU_REF_EINVAL;
}

// splitmix64 stream (reading A15): u = (next() >> 11) * 2^-53
static inline uint64_t splitmix64_next(uint64_t& s) {
  uint64_t z = (s += 0x9E3779B97F4A7C15ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

extern "C" int cosenu_ref_init(cosenu_ref_t* h, uint64_t seed, double sigma_nu, double sigma_nubar,
                               double alpha, double pert_amp, int pert_kind) {
  if (!h) return COSENU_REF_EINVAL;
  if (!(sigma_nu > 0) || !(sigma_nubar > 0) || !(alpha >= 0) || pert_kind < 0 || pert_kind > 2) {
    h->err = "cosenu_ref_init: invalid argument"; return COSENU_REF_EINVAL;
  }
  const int nv = h->nv; const int64_t nz = h->nz;
  // Eq. (20), discretely normalised: sum_j g_j dv = 1 (reading A14); g_bar carries alpha
  std::vector<double> g(nv), gb(nv);
  double sg = 0, sgb = 0;
  for (int j = 0; j < nv; ++j) {
    g[j] = std::exp(-(h->v[j] - 1.0) * (h->v[j] - 1.0) / (2.0 * sigma_nu * sigma_nu));
    gb[j] = std::exp(-(h->v[j] - 1.0) * (h->v[j] - 1.0) / (2.0 * sigma_nubar * sigma_nubar));
    sg += h->wq[j] * g[j]; sgb += h->wq[j] * gb[j];
  }
  for (int j = 0; j < nv; ++j) { g[j] = g[j] / (sg * h->dv); gb[j] = alpha * (gb[j] / (sgb * h->dv)); }
  const double two_pi = 6.283185307179586476925286766559;
  std::vector<double> pr(nz), pi(nz), dd(nz, 1.0);  // perturbation (Re, Im) and ee-xx factor per z
  uint64_t s = seed;
  if (pert_kind == 0) {         // iid uniform phase per z
    for (int64_t i = 0; i < nz; ++i) {
      const double u = (double)(splitmix64_next(s) >> 11) * (1.0 / 9007199254740992.0);
      pr[i] = pert_amp * std::cos(two_pi * u); pi[i] = pert_amp * std::sin(two_pi * u);
    }
  } else if (pert_kind == 1) {  // band-limited: K = 16 lowest modes with seeded phases
    const int K = 16; double ph[K];
    for (int q = 0; q < K; ++q) ph[q] = two_pi * ((double)(splitmix64_next(s) >> 11) * (1.0 / 9007199254740992.0));
    for (int64_t i = 0; i < nz; ++i) {
      double a = 0, b = 0;
      for (int q = 0; q < K; ++q) {
        const double arg = two_pi * (double)(q + 1) * (double)i / (double)nz + ph[q];
        a += std::cos(arg); b += std::sin(arg);
      }
      pr[i] = pert_amp * a / 4.0; pi[i] = pert_amp * b / 4.0;  // 1/sqrt(K)
    }
  } else {                      // Eq. (21): eps(z) = amp exp(-z^2/50), centred at L/2
    for (int64_t i = 0; i < nz; ++i) {
      const double zc = (h->scheme == COSENU_REF_FV_WENO7 ? (i + 0.5) : (double)i) * h->dz - 0.5 * h->L;
      const double e = pert_amp * std::exp(-zc * zc / 50.0);
      pr[i] = 0.5 * e; pi[i] = 0.0; dd[i] = std::sqrt(1.0 - e * e);
    }
  }
  for (int64_t i = 0; i < nz; ++i)
    for (int j = 0; j < nv; ++j) {
      h->y[idx(h, 0, i, j)] = g[j] * 0.5 * (1.0 + dd[i]);  h->y[idx(h, 1, i, j)] = g[j] * 0.5 * (1.0 - dd[i]);
      h->y[idx(h, 2, i, j)] = g[j] * pr[i];                h->y[idx(h, 3, i, j)] = g[j] * pi[i];
      h->y[idx(h, 4, i, j)] = gb[j] * 0.5 * (1.0 + dd[i]); h->y[idx(h, 5, i, j)] = gb[j] * 0.5 * (1.0 - dd[i]);
      h->y[idx(h, 6, i, j)] = gb[j] * pr[i];               h->y[idx(h, 7, i, j)] = gb[j] * pi[i];
    }
  h->t = 0; h->step = 0; h->have_state = true;
  take_references(h);
  return COSENU_REF_OK;
}

extern "C" int cosenu_ref_set_state(cosenu_ref_t* h, const double* host_state, double t) {
  if (!h || !host_state) return COSENU_REF_EINVAL;
  std::memcpy(h->y.data(), host_state, sizeof(double) * h->y.size());
  h->t = t; h->step = 0; h->have_state = true;
  take_references(h);
  return COSENU_REF_OK;
}

extern "C" int cosenu_ref_step(cosenu_ref_t* h, int64_t n) {
  if (!h || n < 0) return COSENU_REF_EINVAL;
  if (!h->have_state) { h->err = "no state: call init or set_state first"; return COSENU_REF_ESTATE; }
  for (int64_t s = 0; s < n; ++s) rk4_step(h);
  return COSENU_REF_OK;
}

extern "C" int cosenu_ref_get_state(cosenu_ref_t* h, double* out) {
  if (!h || !out) return COSENU_REF_EINVAL;
  if (!h->have_state) { h->err = "no state"; return COSENU_REF_ESTATE; }
  std::memcpy(out, h->y.data(), sizeof(double) * h->y.size());
  return COSENU_REF_OK;
}

extern "C" int cosenu_ref_rhs(cosenu_ref_t* h, const double* y, double* k) {
  if (!h || !y || !k) return COSENU_REF_EINVAL;
  rhs(h, y, k); return COSENU_REF_OK;
}

extern "C" int cosenu_ref_moments(cosenu_ref_t* h, const double* y, double* out) {
  if (!h || !y || !out) return COSENU_REF_EINVAL;
  moments(h, y, out); return COSENU_REF_OK;
}

extern "C" int cosenu_ref_diagnostics(cosenu_ref_t* h, cosenu_ref_diag_t* d) {
  if (!h || !d) return COSENU_REF_EINVAL;
  if (!h->have_state) { h->err = "no state"; return COSENU_REF_ESTATE; }
  const double* y = h->y.data();
  d->t = h->t; d->step = h->step;
  long double see[2] = {0, 0}, num = 0, den = 0;
  double dpmax = 0, trmax = 0, exmax = 0;
  for (int s = 0; s < 2; ++s)
    for (int64_t i = 0; i < h->nz; ++i)
      for (int j = 0; j < h->nv; ++j) {
        const long double w = h->wq[j];
        see[s] += w * y[idx(h, 4 * s, i, j)];
        const double P = plen(y, h, s, i, j), Pr = h->Pref[s][j];
        if (Pr > 0) { const double dp = std::fabs(P / Pr - 1.0); if (dp > dpmax) dpmax = dp; }  // Eq. (22)
        if (s == 0) { num += w * std::fabs(P - Pr); den += w * Pr; }                                    // Eq. (23)
        const double tr = std::fabs(y[idx(h, 4 * s, i, j)] + y[idx(h, 4 * s + 1, i, j)] - h->P0ref[s][j]);
        if (tr > trmax) trmax = tr;
        const double ex = std::hypot(y[idx(h, 4 * s + 2, i, j)], y[idx(h, 4 * s + 3, i, j)]);
        if (ex > exmax) exmax = ex;
      }
  d->psurv_nu = h->sum_ee0[0] != 0 ? (double)(see[0] / h->sum_ee0[0]) : 0.0;
  d->psurv_nubar = h->sum_ee0[1] != 0 ? (double)(see[1] / h->sum_ee0[1]) : 0.0;
  d->dP_max = dpmax; d->dP_avg = den > 0 ? (double)(num / den) : 0.0;
  m0_vector(h, y, d->M0);                                                         // Eq. (19)
  for (int m = 0; m < 3; ++m) d->dM0[m] = d->M0[m] - h->M0_init[m];
  d->trace_dev_max = trmax; d->ex_abs_max = exmax;
  return COSENU_REF_OK;
}

extern "C" void cosenu_ref_destroy(cosenu_ref_t* h) { delete h; }
extern "C" const char* cosenu_ref_last_error(const cosenu_ref_t* h) { return h ? h->err.c_str() : g_err.c_str(); }
