"""Host-side analysis helpers of the paper's validation runs (no method arithmetic of the hot path).

As printed in the paper:
  e2_norm               Eq. (15),
  kappa                 Eq. (24),  PAPER.md:292:   log[dP_max(N_z,i) / dP_max(N_z,i+1)] / log 2,  N_z,i+1 = 2 N_z,i, fixed dt
  order_of_convergence  Eq. (C.3):   log((E_i+1 - E_i) / (E_i+2 - E_i+1)) / log r, three errors, fixed dt
and the three scans of the conserved-quantity study of Section 5 (Figs. 8-9), driven through
cosenu_init / cosenu_step / cosenu_diagnostics:
  conserved_quantity_scan   N_z varied at fixed C_CFL
  cfl_scan                  C_CFL varied at fixed N_z            ("in the first one we vary the value of C_CFL for each N_z")
  fixed_dt_scan             N_z varied at fixed dt, 1000 iterations, dt such that the largest N_z has C_CFL = 1 (Fig. 9)
Two textbook estimators that are NOT the paper's equations keep honest names: two_grid_order, richardson_ratio.
"""
import numpy as np


def e2_norm(sim, exact):
    """Eq. (15): sqrt( sum_i (u_sim - u_exact)^2 / N )."""
    d = np.asarray(sim, dtype=np.float64) - np.asarray(exact, dtype=np.float64)
    return float(np.sqrt(np.mean(d * d)))


def kappa(dP_max_i, dP_max_ip1):
    """Eq. (24): kappa = log[dP_max(N_z,i) / dP_max(N_z,i+1)] / log 2 for N_z,i+1 = 2 N_z,i at fixed dt.  It is the spatial order
    of convergence while the spatial error dominates, and goes to zero once the time-integration error does."""
    return float(np.log(dP_max_i / dP_max_ip1) / np.log(2.0))


def order_of_convergence(E_i, E_ip1, E_ip2, ratio=2.0):
    """Eq. (C.3): alpha = log((E_i+1 - E_i) / (E_i+2 - E_i+1)) / log r from the errors on three grids whose spacing shrinks by
    r each time at one and the same dt: the constant C_t dt^beta of Eq. (C.2) cancels in the differences."""
    return float(np.log((E_ip1 - E_i) / (E_ip2 - E_ip1)) / np.log(ratio))


def two_grid_order(err_coarse, err_fine, ratio=2.0):
    """log(err_coarse / err_fine) / log r: the observed order from the errors against a KNOWN solution on two grids (not an
    equation of the paper; used for the advection tests of Section 4.1, where the exact solution is the shifted profile)."""
    return float(np.log(err_coarse / err_fine) / np.log(ratio))


def richardson_ratio(q_coarse, q_mid, q_fine):
    """|q_coarse - q_mid| / |q_mid - q_fine| for a quantity on three successively refined grids: -> r^p for a scheme of order p
    (self-convergence without an exact solution; not an equation of the paper)."""
    den = abs(q_mid - q_fine)
    return float(abs(q_coarse - q_mid) / den) if den > 0 else float("inf")


def _run(make_sim, nz, L, dt, nsteps, seed, pert_amp, pert_kind):
    sim = make_sim(nz, L, dt)
    sim.init(seed, pert_amp=pert_amp, pert_kind=pert_kind)
    sim.step(int(nsteps))
    d = sim.diagnostics()
    sim.close()
    dz = L / nz
    return {"nz": nz, "dz": dz, "dt": dt, "cfl": dt / dz, "steps": int(nsteps), "t": d["t"], "dP_max": d["dP_max"],
            "dP_avg": d["dP_avg"], "dM0_3": d["dM0"][2], "dM0_max": max(abs(x) for x in d["dM0"]), "psurv_nu": d["psurv_nu"]}


def conserved_quantity_scan(make_sim, nz_list, t_end, cfl=0.4, L=None, seed=1, pert_amp=1e-6, pert_kind=0):
    """Fig. 8, along N_z: for every nz run to t_end at dt = cfl * dz and record the deviations of the conserved quantities
    (Eqs. 22, 23 and Eq. 19).  make_sim(nz, L, dt) -> a binding.Cosenu-like object."""
    rows = []
    for nz in nz_list:
        Lz = float(L if L is not None else nz)
        dt = cfl * Lz / nz
        rows.append(_run(make_sim, nz, Lz, dt, round(t_end / dt), seed, pert_amp, pert_kind))
    return rows


def cfl_scan(make_sim, nz, cfl_list, t_end, L, seed=1, pert_amp=1e-2, pert_kind=2):
    """Fig. 8, along C_CFL: one N_z, dt = C_CFL dz for every C_CFL of the list, all runs to the same t_end."""
    rows = []
    for cfl in cfl_list:
        dt = cfl * float(L) / nz
        rows.append(_run(make_sim, nz, float(L), dt, round(t_end / dt), seed, pert_amp, pert_kind))
    return rows


def fixed_dt_scan(make_sim, nz_list, L, nsteps=1000, seed=1, pert_amp=1e-2, pert_kind=2):
    """Fig. 9 (App. C): N_z doubles along nz_list, dt is the same for all of them and such that the largest N_z
    has C_CFL = 1; `nsteps` iterations (the paper: 1000).  Returns the rows and kappa (Eq. 24) between successive N_z."""
    nz_list = list(nz_list)
    assert all(b == 2 * a for a, b in zip(nz_list[:-1], nz_list[1:])), "N_z,i+1 = 2 N_z,i (Eq. 24)"
    dt = float(L) / max(nz_list)
    rows = [_run(make_sim, nz, float(L), dt, nsteps, seed, pert_amp, pert_kind) for nz in nz_list]
    kap = [kappa(a["dP_max"], b["dP_max"]) for a, b in zip(rows[:-1], rows[1:])]
    return rows, kap


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
