"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no stencil, no Hamiltonian, no RK): it
only builds initial states in the canonical host layout  state[8][nz][nv]
(c0=rho_ee, c1=rho_xx, c2=Re rho_ex, c3=Im rho_ex, c4..c7 = same for rho_bar)
and names the five BASELINE.json workloads.  Recipe:

* v-grid: bin centres v_j = -1 + (j + 1/2) 2/nv.
* angular distributions, Eq. (20): g(v) ~ exp(-(v-1)^2 / 2 sigma^2), normalised so
  that sum_j g_j dv = 1; g_bar likewise, then multiplied by alpha = 0.9.
* perturbation: rho_ex = amp * g_j * exp(i phi_i), phi_i = 2 pi u_i, u_i the splitmix64(seed)
  stream (>> 11, * 2^-53) in z order; the same phase for nu and nubar (BASELINE cfg 0).
"""
import numpy as np

_MASK = (1 << 64) - 1


def splitmix64_uniform(seed: int, n: int) -> np.ndarray:
    """n doubles in [0,1) from the splitmix64 stream started at `seed` (pure-integer generator).

    splitmix64's state after i+1 draws is seed + (i+1)*gamma mod 2^64, so the stream vectorises.
    """
    with np.errstate(over="ignore"):
        i = np.arange(1, n + 1, dtype=np.uint64)
        z = np.uint64(seed & _MASK) + i * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


MIDPOINT, TRAPEZOID, SIMPSON = 0, 1, 2


def v_grid(nv: int, quadrature: int = MIDPOINT) -> np.ndarray:
    """Beam velocities: bin centres or, for the trapezoid / Simpson variants of the FD
    implementation, fixed-width vertex-centred points over [-1, 1]."""
    if quadrature == MIDPOINT:
        return -1.0 + (np.arange(nv) + 0.5) * (2.0 / nv)
    return -1.0 + np.arange(nv) * (2.0 / (nv - 1))


def v_weights(nv: int, quadrature: int = MIDPOINT):
    """(dv, w): int f dv ~ dv * sum_j w_j f(v_j)."""
    if quadrature == MIDPOINT:
        return 2.0 / nv, np.ones(nv)
    w = np.ones(nv)
    if quadrature == TRAPEZOID:
        w[0] = w[-1] = 0.5
    else:
        assert nv % 2 == 1 and nv >= 3
        w[:] = np.where(np.arange(nv) % 2 == 1, 4.0 / 3.0, 2.0 / 3.0)
        w[0] = w[-1] = 1.0 / 3.0
    return 2.0 / (nv - 1), w


def angular_distributions(nv: int, sigma_nu=0.6, sigma_nubar=0.5, alpha=0.9, quadrature: int = MIDPOINT):
    v = v_grid(nv, quadrature)
    dv, w = v_weights(nv, quadrature)
    g = np.exp(-(v - 1.0) * (v - 1.0) / (2.0 * sigma_nu * sigma_nu))
    gb = np.exp(-(v - 1.0) * (v - 1.0) / (2.0 * sigma_nubar * sigma_nubar))
    # sequential sums (same order as the C generators) so all three agree to the last bit
    sg = 0.0
    sgb = 0.0
    for j in range(nv):
        sg += w[j] * g[j]
        sgb += w[j] * gb[j]
    g = g / (sg * dv)
    gb = alpha * (gb / (sgb * dv))
    return g, gb


def fast_conversion_state(nz, nv, seed, pert_amp=1e-6, sigma_nu=0.6, sigma_nubar=0.5, alpha=0.9,
                          quadrature: int = MIDPOINT):
    """BASELINE configs 0, 2, 3, 4: z-homogeneous g, g_bar with a seeded random-phase rho_ex."""
    g, gb = angular_distributions(nv, sigma_nu, sigma_nubar, alpha, quadrature)
    phi = 2.0 * np.pi * splitmix64_uniform(seed, nz)
    pr = pert_amp * np.cos(phi)
    pi = pert_amp * np.sin(phi)
    st = np.zeros((8, nz, nv))
    st[0] = g[None, :]
    st[2] = pr[:, None] * g[None, :]
    st[3] = pi[:, None] * g[None, :]
    st[4] = gb[None, :]
    st[6] = pr[:, None] * gb[None, :]
    st[7] = pi[:, None] * gb[None, :]
    return st


def vacuum_check_state(nz, nv, seed, mod_amp=0.1, mod_k=4, pert_amp=1e-3):
    """BASELINE config 1: rho_ee = g (1 + 0.1 sin(2 pi k z/L)), rho_ex from the seeded phase field."""
    g, gb = angular_distributions(nv)
    phi = 2.0 * np.pi * splitmix64_uniform(seed, nz)
    mod = 1.0 + mod_amp * np.sin(2.0 * np.pi * mod_k * np.arange(nz) / nz)
    st = np.zeros((8, nz, nv))
    st[0] = mod[:, None] * g[None, :]
    st[2] = (pert_amp * np.cos(phi))[:, None] * g[None, :]
    st[3] = (pert_amp * np.sin(phi))[:, None] * g[None, :]
    st[4] = mod[:, None] * gb[None, :]
    st[6] = (pert_amp * np.cos(phi))[:, None] * gb[None, :]
    st[7] = (pert_amp * np.sin(phi))[:, None] * gb[None, :]
    return st


def random_state(nz, nv, seed, scale=1.0):
    """Generic O(scale) random state (all 8 components random): for RHS / moment parity tests."""
    u = splitmix64_uniform(seed, 8 * nz * nv).reshape(8, nz, nv)
    return scale * (u - 0.5)


def smooth_random_state(nz, nv, seed, modes=3):
    """Smooth-in-z random state: a few low Fourier modes per (component, v) with seeded amplitudes."""
    u = splitmix64_uniform(seed, 8 * nv * (2 * modes + 1)).reshape(8, nv, 2 * modes + 1)
    z = np.arange(nz) / nz
    st = np.zeros((8, nz, nv))
    for m in range(modes):
        st += (u[:, None, :, 2 * m] - 0.5) * np.cos(2 * np.pi * (m + 1) * z)[None, :, None]
        st += (u[:, None, :, 2 * m + 1] - 0.5) * np.sin(2 * np.pi * (m + 1) * z)[None, :, None]
    st += u[:, None, :, 2 * modes]
    return st


# The five BASELINE.json workloads.  dz = 1, dt = 0.4 dz.
FD4_KO3, FV_WENO7 = 0, 1
CONFIGS = {
    "cfg0": dict(scheme=FD4_KO3, nz=1024, nv=16, L=1024.0, dt=0.4, omega=0.0, theta=0.0, mu=1.0,
                 steps=500, seed=12866, kind="fast"),
    "cfg1": dict(scheme=FD4_KO3, nz=4096, nv=64, L=4096.0, dt=0.4, omega=1.0, theta=0.1, mu=0.0,
                 steps=2000, seed=12867, kind="vacuum"),
    "cfg2": dict(scheme=FV_WENO7, nz=32768, nv=128, L=32768.0, dt=0.4, omega=0.0, theta=0.0, mu=1.0,
                 steps=5000, seed=12868, kind="fast"),
    "cfg3": dict(scheme=FD4_KO3, nz=131072, nv=256, L=131072.0, dt=0.4, omega=0.0, theta=0.0, mu=1.0,
                 steps=200, seed=12869, kind="fast"),
    "cfg4": dict(scheme=FV_WENO7, nz=262144, nv=512, L=262144.0, dt=0.4, omega=1e-2, theta=0.01, mu=1.0,
                 steps=100, seed=12870, kind="fast"),
}


def config_state(name, nz=None):
    """Initial state of a named workload (optionally with nz reduced, for bounded CPU samples)."""
    c = CONFIGS[name]
    n = c["nz"] if nz is None else nz
    if c["kind"] == "vacuum":
        return vacuum_check_state(n, c["nv"], c["seed"])
    return fast_conversion_state(n, c["nv"], c["seed"])
