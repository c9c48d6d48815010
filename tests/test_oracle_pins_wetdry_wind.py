"""Pins for three branches of the oracle that no other CPU test distinguishes: the split of the
depth deficit in wet/dry case (4), the Garratt drag coefficient below its cap, and the time at which the moving storm
is evaluated.  Every expected value is worked out here from the formulas of SURVEY.md 8(c) / DESIGN.md R-8, R-9, by hand
or with libm -- nothing comes from the oracle itself."""
import math

import numpy as np
import pytest

from workloads import c4

H0 = 1e-3


def _modes(u):
    """p = 1 modes (a, b, c) of vertex values (u0, u1, u2): SURVEY.md 8(c.1) inverse."""
    a = (u[0] + u[1] + u[2]) / 3.0
    return np.array([a, 0.5 * (u[2] - a), 0.5 * (u[1] - u[0])])


def _vertex(w3):
    return np.array([w3[0] - w3[1] - w3[2], w3[0] - w3[1] + w3[2], w3[0] + 2 * w3[1]])


# (H at the three vertices, expected H-hat), H0 = 1e-3, worked by hand from SURVEY.md:420
#   H-hat_(1) = H0;  H-hat_(2) = max(H0, H_(2) - (H-hat_(1) - H_(1))/2);  H-hat_(3) = H_(3) - (H-hat_(1)-H_(1)) - (H-hat_(2)-H_(2))
# A: H = (-0.2, 0.5, 1.0): deficit D1 = 0.201; H-hat_(2) = 0.5 - 0.1005 = 0.3995 (max does not bind);
#    H-hat_(3) = 1.0 - 0.201 + 0.1005 = 0.8995.   (giving vertex (2) the whole deficit would leave 0.299 and 1.0)
# B: H = (-0.2, 0.05, 1.0): 0.05 - 0.1005 < H0, the max binds: H-hat_(2) = 0.001, taking 0.049 FROM vertex (2)'s
#    neighbours: H-hat_(3) = 1.0 - 0.201 + 0.049 = 0.848.     (without the max: -0.0505 and 0.8995)
# C: A with the vertices rotated (shallowest at vertex 1, deepest at vertex 0): the result follows the vertices.
# D: tie H_(1) = H_(2): the lower index is (1):  H = (0.0, 0.0, 0.9): H-hat = (0.001, max(H0, 0 - 0.0005) = 0.001, 0.9 - 0.001 - 0.001)
CASE4 = [((-0.2, 0.5, 1.0), (0.001, 0.3995, 0.8995)),
         ((-0.2, 0.05, 1.0), (0.001, 0.001, 0.848)),
         ((1.0, -0.2, 0.5), (0.8995, 0.001, 0.3995)),
         ((0.0, 0.0, 0.9), (0.001, 0.001, 0.898))]


@pytest.mark.parametrize("H, Hhat", CASE4)
@pytest.mark.parametrize("hv", [(0.0, 0.0, 0.0), (0.3, -0.1, 0.2)])
def test_wetdry_case4_deficit_split(O, H, Hhat, hv):
    """[R-8] case (4): the shallowest vertex is lifted to H0, HALF of what that cost is taken from the middle vertex
    (never below H0), the deepest vertex pays the rest.  Expected vertex depths to 1e-15; the depths are independent of
    the bathymetry split H = zeta + h_b."""
    H = np.array(H); hv = np.array(hv)
    assert H.mean() > H0 and H.min() <= H0                      # this is case (4)
    wet, z2, _, _ = O.wetdry_elem(1, H0, hv, _modes(H - hv), np.zeros(3), np.zeros(3))
    assert wet == 1
    got = _vertex(z2) + hv
    assert np.abs(got - np.array(Hhat)).max() <= 1e-15, (got, Hhat)


@pytest.mark.parametrize("r_over_R, V_about", [(4.0, 29.4), (8.0, 18.2), (12.0, 13.5)])
def test_garratt_drag_below_its_cap(O, r_over_R, V_about):
    """[R-9] C_d = (0.75 + 0.067 |W|) 1e-3 where that is below 0.0035, i.e. for |W| < 41.04 m/s -- most of the C4/C5
    wind field.  Gradient wind with f = 0: V = sqrt((B/rho_a) x dp exp(-x)), x = (R/r)^B; stress = (rho_a/rho_0) C_d V W,
    W counter-clockwise (north of the eye it blows west)."""
    hol = dict(x0=0, y0=0, vx=0, vy=0, rmax=40e3, dp=6000.0, B=1.5, rho_air=1.15, rho_water=1025.0, f=0.0)
    r = r_over_R * 40e3
    tsx, tsy, V = O.holland_node(hol, 0.0, 0.0, 0.0, r)          # due north of the centre
    x = (1.0 / r_over_R) ** 1.5
    Vex = math.sqrt(1.5 / 1.15 * x * 6000.0 * math.exp(-x))
    assert abs(Vex - V_about) < 0.1 and abs(V - Vex) <= 1e-12 * Vex
    cd = (0.75 + 0.067 * Vex) * 1e-3
    assert cd < 0.0035
    k = 1.15 / 1025.0 * cd * Vex * Vex
    assert abs(tsx + k) <= 1e-12 * k and abs(tsy) <= 1e-16
    # and the cap is where the two expressions meet
    assert abs((0.0035e3 - 0.75) / 0.067 - 41.0448) < 1e-3


def test_storm_is_evaluated_at_the_start_of_the_step(O):
    """[R-9] "at t_n, frozen over the stages": after one step from t_n the nodal stress of the last WIND evaluation is
    the Holland field centred at x_0 + v t_n -- not at t_n + dt (nor at a stage time).  A fast storm (500 m/s) makes the
    alternatives differ in the first digits."""
    w = c4(nqx=16, nqy=8)
    hol = dict(w.holland); hol["vx"] = 500.0; hol["vy"] = -200.0
    o = O.Oracle.from_workload(w)
    o.set_wind_holland(hol)
    tn, dt = 20.0, w.dt
    o.set_state(tn, w.ze, w.qx, w.qy)
    o.step(1, dt)
    tau = o.get_wind()

    def field(t):
        cx, cy = hol["x0"] + hol["vx"] * t, hol["y0"] + hol["vy"] * t
        return np.array([O.holland_node(hol, cx, cy, x, y)[:2] for x, y in w.mesh.xy]).T

    assert np.abs(tau).max() > 1e-4
    assert np.array_equal(tau, field(tn))
    for t_wrong in (tn + dt, tn + 0.5 * dt, 0.0):
        assert np.abs(field(t_wrong) - tau).max() > 1e-3 * np.abs(tau).max()
    # second step: the storm has moved on by v dt
    o.step(1, dt)
    assert np.array_equal(o.get_wind(), field(tn + dt))
