"""Pins for the oracle's second field integrator (DESIGN.md R-INT; "different integration algorithms for
different user-defined fields"; VERDICT r1 "missing" 4): the Dormand-Prince 5(4) pair.  Its orders against the analytic
helix (a wrong coefficient lowers them), the straight-line limit, whole propagations against the helix and against the
step-doubling integrator, the fringe field against scipy's DOP853, boundary landings, and a shower."""
import ctypes as C
import math

import numpy as np
import pytest

from paper_2203_09467_b200 import workloads as W
from test_oracle_geom_field import _helix

DP = C.POINTER(C.c_double)


def _open_problem(emo, B, integrator, fringe=None):
    surfaces = [(W.PX, -1e4), (W.PX, 1e4), (W.PY, -1e4), (W.PY, 1e4), (W.PZ, -1e4), (W.PZ, 1e4)]
    d = dict(materials=[W.PB], surfaces=surfaces,
             volumes=[dict(surf=list(range(6)), sense=[1, -1, 1, -1, 1, -1], material=-1, tally=-1)],
             field=B, physics=W.physics(n_E=16, integrator=integrator))
    if fringe:
        d["field_fringe"] = fringe
    return emo.Problem(d)


def _dp45(emo, P, x, u, kappa, h):
    x1, u1, err = np.zeros(3), np.zeros(3), C.c_double()
    emo.lib().emo_dp45(P.h, x.ctypes.data_as(DP), u.ctypes.data_as(DP), kappa, h, x1.ctypes.data_as(DP),
                       u1.ctypes.data_as(DP), C.byref(err))
    return x1, u1, err.value


@pytest.mark.parametrize("B", [(0.0, 0.0, 4.0), (0.3, -0.2, 0.5)])
def test_orders_of_the_embedded_pair(emo, B):
    """One step against the analytic helix: the advanced solution is of fifth order (local error ~ h^6: halving h
    divides it by 64), the estimate |x_5 - x_4| is the local error of the fourth-order solution (~ h^5: by 32) and
    bounds the true error of the advanced one."""
    P = _open_problem(emo, B, 1)
    Bh = np.array(B) / np.linalg.norm(B)
    kappa = 0.37
    x0, u0 = np.array([1.0, 2.0, 3.0]), np.array([0.6, 0.0, 0.8])
    true, est = [], []
    for h in (0.8, 0.4, 0.2):
        x1, u1, e = _dp45(emo, P, x0, u0, kappa, h)
        xe, ue = _helix(x0, u0, kappa, Bh, h)
        true.append(np.linalg.norm(x1 - xe))
        est.append(e)
        assert abs(np.linalg.norm(u1) - 1) < 1e-15
        assert true[-1] < e
    for k in (0, 1):
        assert 50 < true[k] / true[k + 1] < 80, true
        assert 27 < est[k] / est[k + 1] < 37, est


def test_no_curvature_is_a_straight_line_with_zero_estimate(emo):
    P = _open_problem(emo, (0.0, 0.0, 4.0), 1)
    x0, u0 = np.array([1.0, 2.0, 3.0]), np.array([0.6, 0.0, 0.8])
    x1, u1, e = _dp45(emo, P, x0, u0, 0.0, 7.0)
    assert np.allclose(x1, x0 + 7.0 * u0, rtol=0, atol=4e-15) and np.allclose(u1, u0, rtol=0, atol=1e-16)
    assert e < 1e-15                              # the error weights sum to zero


@pytest.mark.parametrize("B,q", [((0, 1.0, 0), -1), ((0, 0, 4.0), 1), ((0.3, -0.2, 0.5), -1)])
def test_propagation_follows_the_helix_and_the_other_integrator(emo, B, q):
    P1, P0 = _open_problem(emo, B, 1), _open_problem(emo, B, 0)
    Bm = np.linalg.norm(B)
    Bh = np.array(B) / Bm
    kappa = q * 2.99792458 * Bm / 5.0
    x0, u0 = np.array([1.0, -2.0, 0.5]), np.array([0.48, 0.6, 0.64])
    s_max = min(30.0 / abs(kappa), 500.0)
    s, hit, x, u = P1.propagate_field(0, -1, x0, u0, kappa, s_max)
    assert hit == -1 and s == pytest.approx(s_max, rel=1e-13)
    xe, ue = _helix(x0, u0, kappa, Bh, s)
    nsub = s_max * abs(kappa) / 0.05 + 10
    bound = 1e-7 * nsub + 1e-9                    # the estimate (<= field_eps per accepted substep) bounds the local error
    assert np.linalg.norm(x - xe) < bound
    assert np.linalg.norm(u - ue) < 1e-6 + 2 * abs(kappa) * bound
    s0, hit0, xr, ur = P0.propagate_field(0, -1, x0, u0, kappa, s_max)
    assert np.linalg.norm(x - xr) < 2 * bound


def test_fewer_attempts_than_step_doubling_for_the_same_tolerance(emo):
    """What a second integrator is for: on a smooth stretch the fifth-order pair takes longer substeps."""
    L = emo.lib()
    n = {}
    for integ in (0, 1):
        P = _open_problem(emo, (0.0, 0.0, 4.0), integ)
        x, u = np.array([1.0, -2.0, 0.5]), np.array([0.48, 0.6, 0.64])
        surf, hit, ns = C.c_int(-1), C.c_int(-1), C.c_int(0)
        L.emo_propagate_field_n.restype = C.c_double
        L.emo_propagate_field_n.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int), DP, DP, C.c_double, C.c_double,
                                            C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.emo_propagate_field_n(P.h, 0, C.byref(surf), x.ctypes.data_as(DP), u.ctypes.data_as(DP), 2.4, 60.0, C.byref(hit), C.byref(ns))
        n[integ] = ns.value
    assert n[1] < n[0], n


def test_fringe_trajectory_against_scipy(emo):
    """As test_fringe_trajectory_against_an_independent_integrator, for integrator 1: the field at the stage positions."""
    from scipy.integrate import solve_ivp
    desc, _ = W.get(6, 4)
    P = emo.Problem(dict(desc, physics=dict(desc["physics"], integrator=1)))
    z0, a, Bmag = desc["field_fringe"][0], desc["field_fringe"][1], 4.0
    E = 50.0
    kappa = -2.99792458 * Bmag / math.sqrt(E * (E + 2 * 0.51099895))

    def rhs(s, y):
        x, u = y[:3], y[3:]
        f = 1.0 / (1.0 + math.exp((abs(x[2]) - z0) / a))
        fp = -math.copysign(1.0, x[2]) * f * (1 - f) / a if x[2] != 0 else 0.0
        return np.concatenate([u, kappa * np.cross(u, np.array([-0.5 * x[0] * fp, -0.5 * x[1] * fp, f]))])
    x = np.array([0.5, 0.2, 60.0])
    u = np.array([0.03, 0.02, 1.0])
    u /= np.linalg.norm(u)
    ref = solve_ivp(rhs, (0, 80.0), np.concatenate([x, u]), method="DOP853", rtol=1e-12, atol=1e-14)
    s, hit, xo, uo = P.propagate_field(P.locate(x), -1, x, u, kappa, 80.0)
    assert hit == -1 and s == pytest.approx(80.0, rel=1e-13)
    assert np.linalg.norm(xo - ref.y[:3, -1]) < 2e-5 and np.linalg.norm(uo - ref.y[3:, -1]) < 1e-6


def test_boundary_landings_and_cells(emo):
    """Random charged steps in the 4 T barrel with integrator 1: every step ends inside its cell or ON the surface it
    reports (within the landing tolerance), as for the step doubling (test_field_steps_never_leave_their_cell)."""
    import states
    desc, _ = W.get(4, 4)
    desc = dict(desc, physics=dict(desc["physics"], integrator=1))
    P = emo.Problem(desc)
    n = 3000
    tr = states.random_states(emo, P, desc, n, seed=77)
    res = P.step_batch(tr, 4)
    surf_v = [v for (_, v) in desc["surfaces"]]
    surf_t = [t for (t, _) in desc["surfaces"]]
    n_field = n_land = 0
    for t, r in zip(tr, res):
        if t.ptype == 0 or r.n_sub == 0:
            continue
        n_field += 1
        x = np.array(r.trk.x[:])
        if r.action == 3 and r.trk.alive:
            S = r.trk.surf
            f = (math.hypot(x[0], x[1]) - surf_v[S]) if surf_t[S] == W.CZ else x[surf_t[S]] - surf_v[S]
            assert abs(f) < 3e-7, (S, f)
            n_land += 1
        elif r.trk.alive:
            assert P.locate(x) == r.trk.vol
    assert n_field > 500 and n_land > 100


def test_shower_in_a_field_with_either_integrator(emo):
    """Config 3 (calorimeter in 1 T), 12 primaries: the histories are keyed by ids and steps, the two integrators land
    within 1e-7 cm of each other, so nearly every history is the same: energy closes, the layer profile agrees to a
    percent of its maximum, and the substep counts differ."""
    desc, prim = W.config3(12)
    a = emo.Problem(desc).transport(prim, 3)
    b = emo.Problem(dict(desc, physics=dict(desc["physics"], integrator=1))).transport(prim, 3)
    for r in (a, b):
        assert r["edep"].sum() + r["escaped"] + r["looper"] == pytest.approx(r["E_in"], rel=1e-9)
    assert np.max(np.abs(a["edep"] - b["edep"])) < 0.02 * a["edep"].max()
    assert abs(int(a["steps"].sum()) - int(b["steps"].sum())) < 0.01 * a["steps"].sum()
