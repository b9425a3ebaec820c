"""Hand-computed expectations for outputs of the diagnostics (Eqs. 22, 23) and of the seeded initial
states (Eq. 21) -- shared by the oracle pins (tests/test_oracle_pins.py) and by the GPU tests, which assert
the SAME literal numbers through cosenu_diagnostics / cosenu_init.  No formula of the method is evaluated here: the planted
state is a table of numbers and every expectation below is a literal, derived in the comment next to it.
"""
import numpy as np

NZ, NV = 16, 2
L, DT = 8.0, 0.1


def planted_state():
    """nz = 16, nv = 2.  |P| = |rho_ee - rho_xx| everywhere except one cell with an off-diagonal part.

    nu:    rho_ee = g = (0.3, 1.7) on every row, except row 5: g (1 + delta), delta = (0.5, 0.1).
    nubar: rho_ee = gbar = (0.5, 0.9) on every row, except beam 0 at row 9: 0.5 * 1.8;
           and rhobar_ex = 0.03 - 0.04 i at (row 2, beam 1)   =>   |rhobar_ex| = 0.05 there.
    """
    st = np.zeros((8, NZ, NV))
    st[0, :, 0], st[0, :, 1] = 0.3, 1.7
    st[0, 5, 0], st[0, 5, 1] = 0.3 * 1.5, 1.7 * 1.1
    st[4, :, 0], st[4, :, 1] = 0.5, 0.9
    st[4, 9, 0] = 0.5 * 1.8
    st[6, 2, 1], st[7, 2, 1] = 0.03, -0.04
    return st


# Reference of a beam = z-mean of |P| at the time the state is set (reading R1).
#   nu beam j:  |P|_0 = g_j (1 + delta_j / 16)   ->   0.3 * 1.03125 = 0.309375,  1.7 * 1.00625 = 1.710625
# Eq. (23), <dP> = sum_{z,v} | |P_nu| - |P_nu|_0 | / sum_{z,v} |P_nu|_0   (|P| carries the weight g_v of the paper's integral):
#   one row is off by g delta (1 - 1/16), fifteen rows by g delta / 16   ->   per beam 2 g delta 15/16
#   numerator   2 * 15/16 * (0.3 * 0.5 + 1.7 * 0.1) = 1.875 * 0.32 = 0.6
#   denominator 16 * (0.309375 + 1.710625) = 16 * 2.02 = 32.32
DP_AVG = 0.6 / 32.32            # = 0.018564356435643567 (a mean of |dP| that ignores the weights g_v, or one normalised by the cell count, gives another number)
# Eq. (22), max over both species of | |P| / |P|_0 - 1 |: nubar beam 0, row 9: 0.9 / (0.5 * (1 + 0.8/16)) - 1 = 1.8/1.05 - 1
DP_MAX = 0.7142857142857142
# max | (rho_ee + rho_xx) - z-mean_0 |: nubar beam 0, row 9: 0.9 - 0.525 = 0.375 (nu: 0.140625 and 0.159375)
TRACE_DEV_MAX = 0.375
EX_ABS_MAX = 0.05               # sqrt(0.03^2 + 0.04^2)


def check_planted_diagnostics(d):
    assert abs(d["dP_avg"] - DP_AVG) <= 1e-15, d["dP_avg"]
    assert abs(d["dP_max"] - DP_MAX) <= 1e-15, d["dP_max"]
    assert abs(d["trace_dev_max"] - TRACE_DEV_MAX) <= 1e-15, d["trace_dev_max"]
    assert abs(d["ex_abs_max"] - EX_ABS_MAX) <= 1e-16, d["ex_abs_max"]
    assert abs(d["psurv_nu"] - 1.0) <= 1e-15 and abs(d["psurv_nubar"] - 1.0) <= 1e-15     # ratio to itself at t = 0


# ---- Eq. (21): eps(z) = amp exp(-(z - L/2)^2 / 50).  amp = 0.3; offsets 0, +-5, +-10 from the centre of the box.
E21_AMP = 0.3
E21_EPS_OVER_AMP = {0: 1.0, 5: 0.6065306597126334, 10: 0.1353352832366127}          # 1, e^{-1/2}, e^{-2}
E21_ROOT = {0: 0.9539392014169457, 5: 0.9833060816930658, 10: 0.9991754563138618}    # sqrt(1 - eps^2)
# grids on which those offsets are grid points: FD (z_i = i dz, reading A13): nz = 40, dz = 5 -> z_i - L/2 = 5 (i - 20);
#                                               FV (cell centres):            nz = 41, dz = 5 -> (i + 1/2) 5 - 102.5 = 5 (i - 20)
E21_GRID = {0: (40, 200.0), 1: (41, 205.0)}     # scheme -> (nz, L)


def check_eq21_state(st, scheme):
    """st: (8, nz, nv) produced by init(pert_kind = 2, pert_amp = 0.3) on E21_GRID[scheme]."""
    g, gb = st[0] + st[1], st[4] + st[5]
    assert np.max(np.abs(g - g[0])) <= 1e-15 and np.max(np.abs(gb - gb[0])) <= 1e-15   # rho_ee + rho_xx = g(v) on every row
    for off, e in E21_EPS_OVER_AMP.items():
        for sgn in (+1, -1):
            i = 20 + sgn * (off // 5)
            for (ee, xx, re, im, gg) in ((st[0], st[1], st[2], st[3], g[0]), (st[4], st[5], st[6], st[7], gb[0])):
                assert np.max(np.abs(re[i] - gg * 0.5 * E21_AMP * e)) <= 2e-16 * np.max(gg), (off, sgn)    # Eq. (21c)
                assert np.all(im[i] == 0.0)
                assert np.max(np.abs((ee[i] - xx[i]) - gg * E21_ROOT[off])) <= 4e-16 * np.max(gg)          # Eq. (21a) - (21b)
    # far from the centre the seed is gone: exp(-95^2/50) underflows nothing but is < 1e-78
    assert np.max(np.abs(st[2][1])) < 1e-70


def check_band_limited(st, amp):
    """pert_kind = 1: rho_ex(z) / g = amp/4 * sum of 16 unit phasors of wavenumbers 1..16 -> its DFT along z has exactly 16
    non-zero bins, k = 1..16, each of magnitude amp/4 (numpy's FFT is the independent check)."""
    nz = st.shape[1]
    g = st[0][0] + st[1][0]
    j = int(np.argmax(g))
    f = (st[2][:, j] + 1j * st[3][:, j]) / g[j]
    F = np.fft.fft(f) / nz
    mag = np.abs(F)
    assert np.max(np.abs(mag[1:17] - amp / 4.0)) <= 1e-14 * amp
    rest = np.concatenate([mag[:1], mag[17:]])
    assert np.max(rest) <= 1e-14 * amp
