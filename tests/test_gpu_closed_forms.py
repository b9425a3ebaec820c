"""The CUDA path against what the paper and the mathematics fix, WITHOUT the oracle in between: the discrete
closed form of the linear (mu = 0) system (this is BASELINE config 1's check at full
length), Eq. (17) with the printed 0.076, and the convergence orders of PAPER.md:164."""
import numpy as np
import pytest

from paper_2203_12866_b200 import analysis, inputs
from test_oracle_pins import fd_ko_symbol, linear_closed_form, weno_linear_symbol

pytestmark = pytest.mark.gpu
FD, FV = 0, 1


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2203_12866_b200 import binding
    return binding


def test_config1_full_run_discrete_closed_form(B):
    """BASELINE config 1 (vacuum only, 4096 x 64, 2000 steps): exact advection shift + per-mode precession of the
    DISCRETE scheme (circulant FD4+KO3 symbol x rotation, RK4 stability polynomial to the 2000th power)."""
    c = inputs.CONFIGS["cfg1"]
    st = inputs.config_state("cfg1")
    g = B.Cosenu(c["nz"], c["nv"], c["L"], c["dt"], c["omega"], c["theta"], c["mu"], c["scheme"])
    g.set_state(st)
    g.step(c["steps"])
    got = g.get_state()
    g.close()
    want = linear_closed_form(st, c["steps"], c["dt"], c["omega"], c["theta"],
                              fd_ko_symbol(c["nz"], c["nv"], c["L"] / c["nz"], 0.1))
    assert np.max(np.abs(got - want)) <= 2e-12
    # the loose, continuous version: rho_ee of every beam is the initial modulation shifted by v t (KO damps the
    # k = 4 mode by < 1e-9 here), up to the precession that mixes ee and xx with amplitude sin^2(2 theta)
    tr = got[0] + got[1]
    t = c["steps"] * c["dt"]
    z = np.arange(c["nz"]) * (c["L"] / c["nz"])
    v = inputs.v_grid(c["nv"])
    gnu, _ = inputs.angular_distributions(c["nv"])
    shifted = gnu[None, :] * (1.0 + 0.1 * np.sin(2 * np.pi * 4 * (z[:, None] - v[None, :] * t) / c["L"]))
    assert np.max(np.abs(tr - shifted)) <= 1e-6


def test_weno_linear_limit_closed_form_gpu(B):
    nz, nv, dt, nsteps = 256, 40, 0.4, 300
    st = inputs.random_state(nz, nv, 79)
    g = B.Cosenu(nz, nv, float(nz), dt, 1.0, 0.1, 0.0, FV, weno_eps=1e30)
    g.set_state(st); g.step(nsteps)
    want = linear_closed_form(st, nsteps, dt, 1.0, 0.1, weno_linear_symbol(nz, nv, 1.0))
    assert np.max(np.abs(g.get_state() - want)) <= 2e-13
    g.close()


@pytest.mark.parametrize("scheme", [FD, FV])
def test_eq17_vacuum_solution_gpu(B, golden, scheme):
    gv = golden("paper_values.txt")
    om = float(gv["omega_vac"]); th = np.deg2rad(float(gv["theta_vac_deg"]))
    nz, nv, dt = 64, 4, 0.05
    sim = B.Cosenu(nz, nv, 64.0, dt, om, th, 0.0, scheme)
    st = np.zeros((8, nz, nv)); st[0] = 1.0; st[4] = 0.7
    sim.set_state(st)
    s2, c2 = np.sin(2 * th), np.cos(2 * th)
    minee = 1.0
    for n in range(1, 281):
        sim.step(5)
        t = 5 * n * dt
        ss = np.sin(om * t / 2) ** 2
        want = [1 - s2 * s2 * ss, s2 * s2 * ss, -s2 * c2 * ss, 0.5 * s2 * np.sin(om * t)]
        if n % 20 == 0:
            y = sim.get_state()
            for c in range(4):
                assert np.allclose(y[c], want[c], rtol=0, atol=2e-10), (n, c)
                assert np.allclose(y[4 + c], 0.7 * want[c], rtol=0, atol=2e-10), (n, c)
        d = sim.diagnostics()
        assert abs(d["psurv_nu"] - want[0]) < 2e-10 and abs(d["psurv_nubar"] - want[0]) < 2e-10
        minee = min(minee, d["psurv_nu"])
    sim.close()
    # the printed minimum of <rho_ee>, to its three printed decimals
    assert abs(minee - float(gv["min_rho_ee_theta37"])) < 5e-4


def _advection_error_gpu(B, scheme, nz, eps_ko=None, weno_eps=None, T=2.0):
    nv, L = 2, 2 * np.pi
    dz = L / nz
    nsteps = int(np.ceil(T / (0.02 * dz))); dt = T / nsteps
    sim = B.Cosenu(nz, nv, L, dt, 0.0, 0.0, 0.0, scheme, eps_ko=eps_ko, weno_eps=weno_eps)
    zl = np.arange(nz) * dz
    if scheme == FV:
        f0 = lambda x: (np.cos(x) - np.cos(x + dz)) / dz     # cell averages of sin (reading A13)
    else:
        f0 = np.sin
    st = np.zeros((8, nz, nv)); st[0] = f0(zl)[:, None]
    sim.set_state(st); sim.step(nsteps)
    y = sim.get_state()[0]
    sim.close()
    v = inputs.v_grid(nv)
    return max(analysis.e2_norm(y[:, j], f0(zl - v[j] * T)) for j in range(nv))


def test_convergence_orders_gpu(B, golden):
    gv = golden("paper_values.txt")
    e = [_advection_error_gpu(B, FD, n, eps_ko=0.0) for n in (16, 32)]
    assert abs(analysis.two_grid_order(*e) - float(gv["order_fd4"])) < 0.25
    e = [_advection_error_gpu(B, FV, n, weno_eps=1e30) for n in (16, 32)]
    assert abs(analysis.two_grid_order(*e) - float(gv["order_weno7"])) < 0.4
    e = [_advection_error_gpu(B, FV, n, weno_eps=1e-6) for n in (16, 32)]
    assert 5.0 < analysis.two_grid_order(*e) < 8.5


def test_conserved_quantity_scan_improves_with_resolution(B):
    """Fig. 8, qualitatively: the |P| deviations of the WENO7 run shrink when dz shrinks at
    fixed physical length and C_CFL; M0 stays conserved to rounding at every resolution."""
    rows = analysis.conserved_quantity_scan(
        lambda nz, L, dt: B.Cosenu(nz, 32, L, dt, 0.0, 0.0, 1.0, FV), [256, 512, 1024], t_end=300.0, L=256.0,
        seed=3, pert_amp=1e-3)
    assert rows[2]["dP_max"] < rows[1]["dP_max"] < rows[0]["dP_max"]
    assert all(r["dM0_max"] <= 1e-11 for r in rows)
    assert analysis.richardson_ratio(rows[0]["dP_avg"], rows[1]["dP_avg"], rows[2]["dP_avg"]) > 1.0


# the fiducial fast-conversion set-up of Section 5: Eq. (21) seed of 1e-2, alpha = 0.9; the domain length is
# not printed: 1200, as in the other fiducial tests
_FID_L, _FID_NV = 1200.0, 64


def test_cfl_scan_fd_is_space_limited_fv_is_not(B):
    """PAPER.md:280, Fig. 8(a,b): "doubling the resolution leads to considerable improvements in the errors for both FD and FV.
    However, changing the value of C_CFL alone while keeping N_z unchanged ... does not affect the errors in the case of FD
    whereas the same improves the numerical accuracy of FV"; panel (c): M0_3 stays at its initial value."""
    cfls = [0.8, 0.4, 0.2]
    res = {}
    for scheme in (FD, FV):
        mk = lambda nz, L, dt: B.Cosenu(nz, _FID_NV, L, dt, 0.0, 0.0, 1.0, scheme)
        for nz in (1000, 2000):
            res[scheme, nz] = analysis.cfl_scan(mk, nz, cfls, t_end=250.0, L=_FID_L)
            assert all(abs(r["dM0_3"]) <= 1e-10 for r in res[scheme, nz])
    for scheme in (FD, FV):
        for a, b in zip(res[scheme, 1000], res[scheme, 2000]):                   # doubling N_z: considerable improvement
            assert b["dP_max"] < 0.2 * a["dP_max"] and b["dP_avg"] < 0.3 * a["dP_avg"], (scheme, a, b)
    for nz in (1000, 2000):                                                      # FD: C_CFL alone changes nothing (within 3 %)
        e = [r["dP_max"] for r in res[FD, nz]]
        assert max(e) / min(e) < 1.03, e
        e = [r["dP_avg"] for r in res[FD, nz]]
        assert max(e) / min(e) < 1.03, e
    e = [r["dP_max"] for r in res[FV, 2000]]                                     # FV: a smaller C_CFL improves the accuracy
    assert e[0] > 3.0 * e[1] and e[1] > e[2], e
    e = [r["dP_max"] for r in res[FV, 1000]]
    assert e[0] > 1.15 * e[1] and e[1] >= 0.99 * e[2], e


def test_fixed_dt_scan_kappa(B):
    """PAPER.md:280-294, Fig. 9: dt fixed such that N_z = 32768 has C_CFL = 1, 1000 iterations.  "For FD, the error decreases
    monotonically as we increase N_z.  For FV, however, the error decreases until a saturation value (= 8962 here), after which
    it stays constant"; kappa (Eq. 24) is about constant for FD, with a value like the order of accuracy of Section 4.1, while
    for FV it "initially increases with the increase in N_z and then quickly approaches zero"."""
    nzs = [512, 1024, 2048, 4096, 8192, 16384, 32768]
    rows, kap = analysis.fixed_dt_scan(lambda nz, L, dt: B.Cosenu(nz, _FID_NV, L, dt, 0.0, 0.0, 1.0, FD), nzs, _FID_L)
    assert rows[-1]["cfl"] == 1.0 and all(r["steps"] == 1000 for r in rows)
    e = [r["dP_max"] for r in rows]
    assert all(b < a for a, b in zip(e[:-1], e[1:])), e                          # monotonic
    assert all(2.5 < k < 4.2 for k in kap), kap                                  # FD4 + third-order KO term: kappa ~ 3 - 3.7
    # Eq. (C.3), three errors at one dt: the same spatial order
    al = [analysis.order_of_convergence(e[i], e[i + 1], e[i + 2]) for i in range(len(e) - 2)]
    assert all(2.5 < a < 4.2 for a in al), al
    rows, kap = analysis.fixed_dt_scan(lambda nz, L, dt: B.Cosenu(nz, _FID_NV, L, dt, 0.0, 0.0, 1.0, FV), nzs, _FID_L)
    e = [r["dP_max"] for r in rows]
    assert kap[0] > 5.0 and kap[0] < kap[1] < kap[2] < 8.0, kap                  # rises towards the scheme's order 7
    assert abs(kap[-1]) < 0.5 and abs(kap[-2]) < 0.5, kap                        # then -> 0: saturation
    nsat = next(r["nz"] for r, k in zip(rows[1:], kap) if abs(k) < 0.5) // 2     # last N_z before the error stops falling
    assert 4096 <= nsat <= 16384, nsat                                           # the paper's run: 8962
    assert e[-1] < 1e-3 * e[2]


@pytest.mark.parametrize("scheme", [FD, FV])
def test_fiducial_run_respects_the_light_cone(B, scheme):
    """The paper's fiducial fast-conversion run (alpha = 0.9, sigma = 0.6 / 0.5, Eq. (21) seed
    eps(z) = 1e-2 exp(-z^2/50), N_z = 2000, N_v = 100, C_CFL = 0.2; the domain length is not printed -- 1200 here):
    "flavor waves ... never cross the light cone" (|v| <= 1).  Inside the cone the instability has grown by orders of
    magnitude; far outside it the off-diagonal elements are still at the level of the seed's Gaussian tail.  Also:
    the beam v_z = 0.99 of Fig. 6 exists (bin centres), and M0 is conserved to rounding."""
    nz, nv, L = 2000, 100, 1200.0
    dz = L / nz
    dt = 0.2 * dz
    g = B.Cosenu(nz, nv, L, dt, 0.0, 0.0, 1.0, scheme)
    g.init(1, pert_amp=1e-2, pert_kind=2)
    st0 = g.get_state()
    t_end = 250.0
    nsteps = int(round(t_end / dt))
    g.step(nsteps)
    st = g.get_state()
    d = g.diagnostics()
    g.close()
    assert abs(inputs.v_grid(nv)[-1] - 0.99) < 1e-15
    zc = (np.arange(nz) + (0.5 if scheme == FV else 0.0)) * dz - 0.5 * L        # the seed is centred at L/2
    gj = st0[0].max(axis=0)                                                      # g_nu(v) (rho_ee + rho_xx at t = 0)
    ex = np.sqrt(st[2] ** 2 + st[3] ** 2) / gj[None, :]                          # |rho_ex| / g
    inside = np.abs(zc) < 0.5 * t_end
    outside = np.abs(zc) > t_end + 60.0                                          # light cone + the seed's own width
    assert outside.sum() > 100
    assert ex[inside].max() > 0.05                                               # the conversion has developed
    assert ex[outside].max() < 1e-9                                              # and has not crossed the cone
    assert max(abs(x) for x in d["dM0"]) <= 1e-10
    assert d["trace_dev_max"] <= 1e-12                                           # 2083 steps of rounding on O(1) traces
    # waves propagate primarily toward +z: more converted flavour on the +z side of the centre
    pz = 1.0 - (st[0] / (st[0] + st[1]))                                         # rho_xx fraction per cell
    assert pz[zc > 0].sum() > pz[zc < 0].sum()


@pytest.mark.parametrize("scheme", [FD, FV])
def test_boxcar_advection_paper_setup(B, scheme):
    """PAPER.md:180-185 at the paper's size and length (N_z = 2000 and 4000, C_CFL = 0.2, v = 0.5, t = 600): max error ~ 0.5,
    unchanged with resolution; E2 drops; Gibbs oscillations for FD only."""
    from test_oracle_pins import boxcar_run, check_boxcar
    mk = lambda nz, nv, L, dt, s: B.Cosenu(nz, nv, L, dt, 0.0, 0.0, 0.0, s)
    check_boxcar([boxcar_run(mk, scheme, nz, T=600.0) for nz in (2000, 4000)], scheme)


def test_fd_without_ko_dissipation_turns_unphysical(B):
    """PAPER.md:269-271 (Fig. 7): in the fiducial run "the FD simulation without dissipation leads to numerical instabilities
    starting at t ~ 800 ... and produces unphysically large values of P_3 > 1", which the Kreiss-Oliger term (eps_KO = 0.1)
    and the FV scheme do not.  P_3 = (rho_ee - rho_xx) / (rho_ee + rho_xx) per cell.  (Domain length not printed: 1200.)"""
    nz, nv, L = 2000, 100, 1200.0
    dz = L / nz
    dt = 0.2 * dz
    worst = {}
    for name, scheme, eps in (("fd_no_ko", FD, 0.0), ("fd_ko", FD, 0.1), ("fv", FV, None)):
        g = B.Cosenu(nz, nv, L, dt, 0.0, 0.0, 1.0, scheme, eps_ko=eps)
        g.init(1, pert_amp=1e-2, pert_kind=2)
        g.step(int(round(800.0 / dt)))
        st = g.get_state()
        g.close()
        worst[name] = max(np.abs((st[0] - st[1]) / (st[0] + st[1])).max(), np.abs((st[4] - st[5]) / (st[4] + st[5])).max())
    assert worst["fd_no_ko"] > 1.0 + 1e-3, worst
    assert worst["fd_ko"] < 1.0 + 1e-6 and worst["fv"] < 1.0 + 1e-6, worst
