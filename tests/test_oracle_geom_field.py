"""Pins for the oracle's geometry and uniform-field propagation (C9)."""
import math

import numpy as np
import pytest

from paper_2203_09467_b200 import workloads as W


def _inside(desc, vol, x):
    """Brute-force point-in-cell test written directly from the surface definitions."""
    for S, sense in zip(desc["volumes"][vol]["surf"], desc["volumes"][vol]["sense"]):
        t, v = desc["surfaces"][S]
        f = x[0] ** 2 + x[1] ** 2 - v * v if t == W.CZ else x[t] - v
        if (1 if f > 0 else -1) != sense:
            return False
    return True


def _march(desc, vol, x, u, smax, ds):
    s = 0.0
    while s < smax:
        if not _inside(desc, vol, x + (s + ds) * u):
            lo, hi = s, s + ds
            for _ in range(60):
                mid = 0.5 * (lo + hi)
                if _inside(desc, vol, x + mid * u):
                    lo = mid
                else:
                    hi = mid
            return 0.5 * (lo + hi)
        s += ds
    return math.inf


@pytest.mark.parametrize("cfg", [1, 2, 4])
def test_distance_against_ray_marching(emo, cfg):
    desc, _ = W.get(cfg, 4)
    P = emo.Problem(desc)
    rng = np.random.default_rng(cfg)
    checked = 0
    for _ in range(300):
        if cfg == 4:
            r = rng.uniform(0, 294); ph = rng.uniform(0, 2 * math.pi)
            x = np.array([r * math.cos(ph), r * math.sin(ph), rng.uniform(-149, 149)])
        elif cfg == 2:
            x = np.array([rng.uniform(-29, 29), rng.uniform(-29, 29), rng.uniform(-9, 49)])
        else:
            x = np.array([rng.uniform(-49, 49), rng.uniform(-49, 49), rng.uniform(1, 99)])
        vol = P.locate(x)
        assert vol >= 0 and _inside(desc, vol, x)
        u = rng.normal(size=3); u /= np.linalg.norm(u)
        d, hit = P.distance(vol, x, u)
        ref = _march(desc, vol, x, u, 700.0, 0.011)
        if math.isfinite(ref) and ref > 0.05:       # marching can step over grazing chords shorter than ds
            assert d == pytest.approx(ref, rel=1e-9, abs=1e-9)
            checked += 1
            # the landing point lies on the reported surface
            t, v = desc["surfaces"][hit]
            y = x + d * u
            f = math.hypot(y[0], y[1]) - v if t == W.CZ else y[t] - v
            assert abs(f) < 1e-9
    assert checked > 200


def test_cylinder_chord_and_on_surface_rules(emo):
    desc, _ = W.config4(4)
    P = emo.Problem(desc)
    R = desc["surfaces"][0][1]          # 5 cm, cell 0 is inside it
    # chord through the axis plane at impact parameter b: length 2 sqrt(R^2 - b^2) / sin(theta)
    for b, uz in ((0.0, 0.0), (3.0, 0.0), (4.9, 0.3)):
        s = math.sqrt(1 - uz * uz)
        x = np.array([-math.sqrt(R * R - b * b), b, 0.0])      # on the cylinder
        u = np.array([s, 0.0, uz])
        d, hit = P.distance(0, x, u, surf=0)
        assert hit == 0 and d == pytest.approx(2 * math.sqrt(R * R - b * b) / s, rel=1e-13)
    # flagged on the cylinder and pointing outwards from the inside cell: immediate re-crossing, d = 0
    d, hit = P.distance(0, np.array([R, 0.0, 0.0]), np.array([1.0, 0.0, 0.0]), surf=0)
    assert (d, hit) == (0.0, 0)
    # outside cell (cell 1 = Si shell between CZ0 and CZ1), flagged on CZ0, moving outwards: CZ0 is skipped
    d, hit = P.distance(1, np.array([R, 0.0, 0.0]), np.array([1.0, 0.0, 0.0]), surf=0)
    assert hit == 1 and d == pytest.approx(0.03, rel=1e-12)
    # parallel to the axis: only the end planes
    d, hit = P.distance(0, np.array([1.0, 1.0, 0.0]), np.array([0.0, 0.0, 1.0]))
    assert hit == 84 and d == pytest.approx(150.0)


def test_straight_track_through_the_calorimeter_stack(emo):
    desc, _ = W.config2(4)
    P = emo.Problem(desc)
    u = np.array([0.05, -0.02, 1.0]); u /= np.linalg.norm(u)
    x = np.array([0.0, 0.0, -0.1]); vol, surf = 100, -1
    path = {}
    seq = []
    for _ in range(300):
        d, hit = P.distance(vol, x, u, surf)
        path[vol] = path.get(vol, 0.0) + d
        x = x + d * u
        nv = P.neighbour(x, u, hit)
        seq.append(vol)
        if nv < 0:
            break
        vol, surf = nv, hit
    assert seq == [100] + list(range(100)) + [101]       # front vacuum, layers 0..99 in order, back vacuum
    for layer in range(100):
        thick = 0.23 if layer % 2 == 0 else 0.57
        assert path[layer] == pytest.approx(thick / u[2], rel=1e-12)
    assert sum(path.values()) == pytest.approx(50.1 / u[2], rel=1e-13)


def test_neighbour_sideways_exit_and_world_escape(emo):
    desc, _ = W.config2(4)
    P = emo.Problem(desc)
    # leave layer 10 through x = +20 -> right vacuum box (103), then through x = +30 -> outside
    x = np.array([20.0, 1.0, 4.1]); u = np.array([1.0, 0.0, 0.0])
    assert P.neighbour(x, u, 105) == 103
    assert P.neighbour(np.array([30.0, 1.0, 4.1]), u, 106) == -1
    # crossing back into the stack from the side box lands in the right layer
    assert P.neighbour(x, -u, 105) == 10      # z = 4.1 lies in Pb_5 = [4.0, 4.23] = volume 10
    # on an edge (also on a z plane): direction decides
    x = np.array([20.0, 0.0, 0.8]); ud = np.array([-0.6, 0.0, 0.8])
    assert P.neighbour(x, ud, 105) == 2
    assert P.neighbour(x, np.array([-0.6, 0.0, -0.8]), 105) == 1


# ---------------- field ----------------

def _helix(x0, u0, kappa, Bhat, s):
    """Analytic solution of du/ds = kappa u x Bhat."""
    Bhat = np.asarray(Bhat, float)
    upar = (u0 @ Bhat) * Bhat
    uperp = u0 - upar
    w = np.cross(uperp, Bhat)
    x = x0 + upar * s + (uperp * math.sin(kappa * s) + w * (1 - math.cos(kappa * s))) / kappa
    u = upar + uperp * math.cos(kappa * s) + w * math.sin(kappa * s)
    return x, u


def _open_problem(emo, B):
    surfaces = [(W.PX, -1e4), (W.PX, 1e4), (W.PY, -1e4), (W.PY, 1e4), (W.PZ, -1e4), (W.PZ, 1e4)]
    d = dict(materials=[W.PB], surfaces=surfaces,
             volumes=[dict(surf=list(range(6)), sense=[1, -1, 1, -1, 1, -1], material=-1, tally=-1)],
             field=B, physics=W.physics(n_E=16))
    return emo.Problem(d)


def test_rk4_doubling_error_estimate(emo):
    import ctypes as C
    L = emo.lib()
    dp = C.POINTER(C.c_double)
    x0 = np.zeros(3); u0 = np.array([0.6, 0.0, 0.8]); Bh = np.array([0.0, 0.0, 1.0])
    kappa = -2.5
    for h in (0.02, 0.05, 0.1):
        x1 = np.zeros(3); u1 = np.zeros(3); err = C.c_double()
        L.emo_rk4_doubling(x0.ctypes.data_as(dp), u0.ctypes.data_as(dp), kappa, Bh.ctypes.data_as(dp), h,
                           x1.ctypes.data_as(dp), u1.ctypes.data_as(dp), C.byref(err))
        xe, ue = _helix(x0, u0, kappa, Bh, h)
        true = np.linalg.norm(x1 - xe)
        assert true <= err.value / 10          # Richardson: the half-step result is ~16x better
        assert abs(np.linalg.norm(u1) - 1) < 1e-15
        assert abs(u1 @ Bh - u0 @ Bh) < 1e-4 * (h * kappa) ** 6 + 1e-15   # pitch: only the RK4 norm drift (renormalised)


@pytest.mark.parametrize("B,q", [((0, 1.0, 0), -1), ((0, 0, 4.0), 1), ((0.3, -0.2, 0.5), -1)])
def test_propagation_follows_the_analytic_helix(emo, B, q):
    P = _open_problem(emo, B)
    Bm = np.linalg.norm(B); Bh = np.array(B) / Bm
    p = 5.0                                     # MeV/c
    kappa = q * 2.99792458 * Bm / p
    x0 = np.array([1.0, -2.0, 0.5]); u0 = np.array([0.48, 0.6, 0.64])
    s_max = 30.0 / abs(kappa) if abs(kappa) * 30 < 200 else 100.0
    s_max = min(s_max, 500.0)
    s, hit, x, u = P.propagate_field(0, -1, x0, u0, kappa, s_max)
    assert hit == -1 and s == pytest.approx(s_max, rel=1e-13)
    xe, ue = _helix(x0, u0, kappa, Bh, s)
    nsub = s_max * abs(kappa) / 0.05 + 10       # crude bound on the number of substeps
    bound = 1e-7 * nsub / 15 + 1e-9             # local error <= eps / 15 per substep
    assert np.linalg.norm(x - xe) < bound
    assert np.linalg.norm(u - ue) < 1e-6 + 2 * abs(kappa) * bound   # a phase error turns u by |kappa| times the arc it costs


def test_radius_of_curvature_1T_1MeV(emo):
    """Pins the curvature constant of emo_step itself (r = 0.33356 cm for p = 1 MeV/c, B = 1 T) to
    something outside the oracle: r = p / (|q| B) in SI units with p = 1e6 eV/c, i.e. r = 1e6 V / (c B) with the
    SI-exact c = 299 792 458 m/s.  An electron of that momentum takes one capped vacuum step of 0.1 cm in a 1 T
    field along z; its direction must have turned by s / r about z, anticlockwise for the negative charge (du/ds =
    kappa u x B, kappa < 0) and clockwise for a positron."""
    r_cm = 1e6 / (299792458.0 * 1.0) * 100.0
    assert r_cm == pytest.approx(0.33356, rel=1e-4)
    surfaces = [(W.PX, -1e4), (W.PX, 1e4), (W.PY, -1e4), (W.PY, 1e4), (W.PZ, -1e4), (W.PZ, 1e4)]
    d = dict(materials=[W.PB], surfaces=surfaces, seed=1,
             volumes=[dict(surf=list(range(6)), sense=[1, -1, 1, -1, 1, -1], material=-1, tally=-1)],
             field=(0.0, 0.0, 1.0), physics=W.physics(n_E=16, vacuum_step=0.1))
    P = emo.Problem(d)
    T = math.sqrt(1.0 + emo.ME ** 2) - emo.ME                 # kinetic energy of p = 1 MeV/c
    for ptype, sign in ((1, +1.0), (2, -1.0)):
        tr = (emo.Track * 1)()
        tr[0].u[:] = [1.0, 0.0, 0.0]
        tr[0].E, tr[0].vol, tr[0].surf, tr[0].ptype, tr[0].alive = T, 0, -1, ptype, 1
        o = P.step_batch(tr, 1)[0]
        assert o.s == pytest.approx(0.1, rel=1e-13) and o.action == 4
        ang = o.s / r_cm
        assert o.trk.u[0] == pytest.approx(math.cos(ang), abs=2e-7)       # RK4 local error 1e-7 cm over a 0.1 cm arc
        assert o.trk.u[1] == pytest.approx(sign * math.sin(ang), abs=2e-7)
        assert abs(o.trk.u[2]) < 1e-15
        # the end point lies on the circle of radius r through the origin, centre (0, sign r, 0)
        assert math.hypot(o.trk.x[0], o.trk.x[1] - sign * r_cm) == pytest.approx(r_cm, rel=1e-6)
    # and the propagator alone, half a turn: the chord is the diameter
    P2 = _open_problem(emo, (0, 0, 1.0))
    kappa = -1.0 / r_cm
    s, hit, x, u = P2.propagate_field(0, -1, np.zeros(3), np.array([1.0, 0.0, 0.0]), kappa, math.pi * r_cm)
    assert np.linalg.norm(x) == pytest.approx(2 * r_cm, rel=1e-6)


def test_weak_field_limit_is_a_straight_line(emo):
    P = _open_problem(emo, (0, 1e-12, 0))
    x0 = np.array([0.0, 0.0, 0.0]); u0 = np.array([0.0, 0.6, 0.8])
    s, hit, x, u = P.propagate_field(0, -1, x0, u0, -1e-15, 50.0)
    assert s == pytest.approx(50.0, rel=1e-13) and np.allclose(x, 50.0 * u0, atol=1e-9) and np.allclose(u, u0, atol=1e-12)


def test_boundary_landing_in_field(emo):
    desc, _ = W.config3(4)
    P = emo.Problem(desc)
    eps = desc["physics"]["field_eps"]
    rng = np.random.default_rng(11)
    n_hit = 0
    for _ in range(200):
        layer = int(rng.integers(0, 100))
        z0, z1 = desc["surfaces"][layer][1], desc["surfaces"][layer + 1][1]
        x0 = np.array([rng.uniform(-5, 5), rng.uniform(-5, 5), rng.uniform(z0 + 1e-3, z1 - 1e-3)])
        u0 = rng.normal(size=3); u0 /= np.linalg.norm(u0)
        p = 10 ** rng.uniform(-0.5, 2)
        kappa = -2.99792458 * 1.0 / p
        s, hit, x, u = P.propagate_field(layer, -1, x0, u0, kappa, 5.0)
        xe, ue = _helix(x0, u0, kappa, np.array([0, 1.0, 0]), s)
        assert np.linalg.norm(x - xe) < 1e-5          # on the true helix
        if hit >= 0:
            n_hit += 1
            t, v = desc["surfaces"][hit]
            assert abs(x[t] - v) <= 2 * eps           # landed within tolerance of the surface
            assert hit in (layer, layer + 1, 104, 105, 108, 109)
        else:
            assert s == pytest.approx(5.0, rel=1e-13) and z0 < x[2] < z1
    assert n_hit > 150


@pytest.mark.parametrize("cfg,n", [(3, 6000), (4, 6000)])
def test_field_steps_never_leave_their_cell(emo, cfg, n):
    """Invariant (C9): a step ends inside or on the boundary of the cell it started in -- a
    boundary may be reached, never passed.  Pins the landing rule |L - d| <= eps: with the one-sided rule
    L - d <= eps a chord end a hair SHORT of a surface was accepted as interior, rounded onto the surface
    unflagged, and the next chord walked through it (seen as end points 7 cm outside the cell)."""
    import states
    desc, _ = W.get(cfg, 4)
    P = emo.Problem(desc)
    tr = states.random_states(emo, P, desc, n, seed=1000 + cfg, ptypes=(1, 2))
    res = P.step_batch(tr, desc["seed"])
    worst = 0.0
    for t, r in zip(tr, res):
        vol = desc["volumes"][t.vol]
        x = r.trk.x
        for S, sense in zip(vol["surf"], vol["sense"]):
            ty, v = desc["surfaces"][S]
            f = (math.hypot(x[0], x[1]) - v) if ty == 3 else (x[ty] - v)
            worst = max(worst, -sense * f)          # > 0: outside this face by that many cm
    assert worst <= 2e-7                             # landing tolerance eps = 1e-7 cm


def test_field_landing_regression_state(emo):
    """The state that exposed the one-sided landing rule: a 4 keV e- in the bottom vacuum box of the
    calorimeter world, B = 1 T along y.  It spirals about y with r = 0.02 cm (two steps end on the substep
    budget, action TRUNC, 4.4 cm of arc each) and must then stop ON the y = -30 cm face (surface 107) and escape."""
    desc, _ = W.get(3, 4)
    P = emo.Problem(desc)
    t = emo.Track()
    t.x[:] = [15.723231344610966, -26.661460451909164, 6.158366420181668]
    t.u[:] = [-0.7636925592807772, -0.26691181033127387, 0.5878194964484071]
    t.E = 0.003987383479174055; t.vol = 104; t.surf = -1; t.ptype = 1; t.alive = 1
    acts = []
    for _ in range(10):
        r = P.step_batch((emo.Track * 1)(t), 3)[0]
        acts.append(r.action)
        assert -30.0 - 1e-7 <= r.trk.x[1] and -20.0 <= r.trk.x[0] <= 20.0 and 0.0 <= r.trk.x[2] <= 40.0   # never outside cell 104
        if not r.trk.alive:
            break
        t = r.trk
    assert acts == [4, 4, 3]
    assert r.trk.surf == 107 and abs(r.trk.x[1] + 30.0) <= 1e-7 and r.escaped == pytest.approx(0.003987383479174055)


# ---------------- non-uniform field: solenoid with a fringe ----------------

def _fringe_problem(emo, z0=100.0, a=15.0):
    desc, _ = W.get(6, 4)
    desc = dict(desc)
    desc["field_fringe"] = (z0, a)
    return emo.Problem(desc)


def test_fringe_field_profile_closed_forms(emo):
    """g(x): on the axis only B_z, equal to 1/2 at |z| = z0 and to the logistic elsewhere; even in z; the radial
    part points outwards where the field falls off (beyond the centre) and div g = 0 by central differences."""
    P = _fringe_problem(emo)
    L = emo.lib()

    def g(x):
        out = np.zeros(3)
        L.emo_field_profile(P.h, emo._dp(np.asarray(x, dtype=np.float64)), emo._dp(out))
        return out
    assert g([0, 0, 100.0]) == pytest.approx([0, 0, 0.5], abs=1e-15)
    assert g([0, 0, -100.0]) == pytest.approx([0, 0, 0.5], abs=1e-15)
    assert g([0, 0, 130.0])[2] == pytest.approx(1.0 / (1.0 + math.exp(2.0)), rel=1e-14)
    assert g([0, 0, 0.0])[2] == pytest.approx(1.0 / (1.0 + math.exp(-100.0 / 15.0)), rel=1e-14)
    a, b = g([3.0, -2.0, 120.0]), g([3.0, -2.0, -120.0])
    assert a[2] == b[2] and a[0] == -b[0] and a[1] == -b[1]
    assert a[0] > 0 and a[1] < 0                                   # field lines open up where B_z decreases
    x0, h = np.array([7.0, -4.0, 95.0]), 1e-4
    div = sum((g(x0 + h * e)[k] - g(x0 - h * e)[k]) / (2 * h) for k, e in enumerate(np.eye(3)))
    assert abs(div) < 1e-9


def test_fringe_integrator_reduces_to_the_uniform_one(emo):
    """With the fringe pushed out to |z| = 1e9 cm the profile is exactly (0, 0, 1) and the stage-position
    integrator must give bit-identical results to the uniform-field one."""
    P = _fringe_problem(emo, z0=1e9, a=1.0)
    L = emo.lib()
    rng = np.random.default_rng(7)
    Bhat = np.array([0.0, 0.0, 1.0])
    for _ in range(50):
        x = rng.normal(0, 50, 3)
        u = rng.normal(0, 1, 3)
        u /= np.linalg.norm(u)
        kappa, h = rng.choice([-1, 1]) * 10 ** rng.uniform(-4, 0), 10 ** rng.uniform(-3, 1)
        x1, u1, x2, u2 = np.zeros(3), np.zeros(3), np.zeros(3), np.zeros(3)
        e1, e2 = emo.C.c_double(), emo.C.c_double()
        L.emo_rk4_doubling(emo._dp(x), emo._dp(u), kappa, emo._dp(Bhat), h, emo._dp(x1), emo._dp(u1), emo.C.byref(e1))
        L.emo_rk4_doubling_map(P.h, emo._dp(x), emo._dp(u), kappa, h, emo._dp(x2), emo._dp(u2), emo.C.byref(e2))
        assert np.array_equal(x1, x2) and np.array_equal(u1, u2) and e1.value == e2.value


def test_fringe_trajectory_against_an_independent_integrator(emo):
    """A 50 MeV electron from the centre of the barrel through the fringe region: the oracle's adaptive RK4
    (inside the vacuum core, no boundary in reach) against scipy's DOP853 at rtol 1e-12 on the same equation
    of motion written out here.  Tolerance: field_eps (1e-7 cm) per accepted substep."""
    from scipy.integrate import solve_ivp
    P = _fringe_problem(emo)
    L = emo.lib()
    z0, a, Bmag = 100.0, 15.0, 4.0
    E = 50.0
    ME = 0.51099895                                                  # MeV
    pm = math.sqrt(E * (E + 2 * ME))
    kappa = -1.0 * 2.99792458 * Bmag / pm

    def rhs(s, y):
        x, u = y[:3], y[3:]
        f = 1.0 / (1.0 + math.exp((abs(x[2]) - z0) / a))
        fp = -math.copysign(1.0, x[2]) * f * (1 - f) / a if x[2] != 0 else 0.0
        g = np.array([-0.5 * x[0] * fp, -0.5 * x[1] * fp, f])
        return np.concatenate([u, kappa * np.cross(u, g)])
    x = np.array([0.5, 0.2, 60.0])
    u = np.array([0.03, 0.02, 1.0])
    u /= np.linalg.norm(u)
    s_max = 80.0                                                     # stays inside r < 5 cm, |z| < 150
    ref = solve_ivp(rhs, (0, s_max), np.concatenate([x, u]), method="DOP853", rtol=1e-12, atol=1e-14)
    xo, uo = x.copy(), u.copy()
    surf = emo.C.c_int(-1)
    hit = emo.C.c_int(-1)
    vol = P.locate(x)
    s = L.emo_propagate_field(P.h, vol, emo.C.byref(surf), emo._dp(xo), emo._dp(uo), kappa, s_max, emo.C.byref(hit))
    assert hit.value == -1 and s == pytest.approx(s_max, rel=1e-13)
    assert np.linalg.norm(xo - ref.y[:3, -1]) < 2e-5                 # ~100 substeps of 1e-7 cm local error
    assert np.linalg.norm(uo - ref.y[3:, -1]) < 1e-6
    # and it differs from the uniform-field trajectory by far more than that (the test sees the fringe)
    Pu = emo.Problem(W.get(4, 4)[0])
    xu, uu = x.copy(), u.copy()
    surf2, hit2 = emo.C.c_int(-1), emo.C.c_int(-1)
    L.emo_propagate_field(Pu.h, vol, emo.C.byref(surf2), emo._dp(xu), emo._dp(uu), kappa, s_max, emo.C.byref(hit2))
    assert np.linalg.norm(xu - xo) > 1e-3
