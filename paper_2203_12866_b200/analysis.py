"""Host-side analysis helpers of the paper's validation runs (no method arithmetic of the hot path).

E2 error norm (Eq. 15), the convergence indicator kappa (Eq. 24) and the
order-of-convergence estimator (Eq. C.3), plus the conserved-quantity scan of Fig. 8
 driven through cosenu_diagnostics.
"""
import numpy as np


def e2_norm(sim, exact):
    """Eq. (15): sqrt( sum_i (u_sim - u_exact)^2 / N )."""
    d = np.asarray(sim, dtype=np.float64) - np.asarray(exact, dtype=np.float64)
    return float(np.sqrt(np.mean(d * d)))


def order_of_convergence(err_coarse, err_fine, ratio=2.0):
    """Eq. (C.3): observed order p from the errors on two grids whose spacing differs by `ratio`."""
    return float(np.log(err_coarse / err_fine) / np.log(ratio))


def kappa(q_coarse, q_mid, q_fine):
    """Eq. (24): kappa = |q_coarse - q_mid| / |q_mid - q_fine| for a quantity computed on three successively
    refined grids; kappa -> 2^p for a scheme of order p (self-convergence, no exact solution needed)."""
    den = abs(q_mid - q_fine)
    return float(abs(q_coarse - q_mid) / den) if den > 0 else float("inf")


def conserved_quantity_scan(make_sim, nz_list, t_end, cfl=0.4, L=None, seed=1, pert_amp=1e-6):
    """Fig. 8-style scan: for every nz run to t_end at dt = cfl * dz and record the deviations of the conserved
    quantities (Eq. 22, 23 and Eq. 19).  make_sim(nz, L, dt) -> a binding.Cosenu-like object."""
    rows = []
    for nz in nz_list:
        Lz = float(L if L is not None else nz)
        dz = Lz / nz
        dt = cfl * dz
        sim = make_sim(nz, Lz, dt)
        sim.init(seed, pert_amp=pert_amp)
        sim.step(int(round(t_end / dt)))
        d = sim.diagnostics()
        rows.append({"nz": nz, "dz": dz, "dt": dt, "t": d["t"], "dP_max": d["dP_max"], "dP_avg": d["dP_avg"],
                     "dM0_max": max(abs(x) for x in d["dM0"]), "psurv_nu": d["psurv_nu"]})
        sim.close()
    return rows


def polarization_norm(state, species=0):
    """|P|(z,v) of Eq. (4) from a canonical state (8, nz, nv): sqrt((ee-xx)^2 + 4 |ex|^2), un-normalised."""
    o = 4 * species
    st = np.asarray(state, dtype=np.float64)
    return np.sqrt((st[o] - st[o + 1]) ** 2 + 4.0 * (st[o + 2] ** 2 + st[o + 3] ** 2))


def dP_map(state, state0, species=0):
    """The map delta P(z, v) = |P|(t) / |P|_0(v) - 1 of Fig. 10, |P|_0(v) = z-mean at t = 0 (the
    reference cosenu_diagnostics uses for Eq. 22); its max |.| over (z,v) and both species is `dP_max`."""
    p0 = polarization_norm(state0, species).mean(axis=0)
    return polarization_norm(state, species) / p0[None, :] - 1.0
