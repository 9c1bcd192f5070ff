"""Pins for the spatial part of the oracle's multiple scattering (DESIGN.md R-MSC2; PAPER.md:111 names Urban /
WentzelVI and prints no formula; VERDICT r1 "What's missing" 1: path-length correction and lateral displacement):
the second transport cross section against a quadrature of the single-scattering law, Lewis' <z> and <x^2 + y^2>
against their plain formulas in 50-digit arithmetic AND against a brute-force collision-by-collision simulation of
the screened Rutherford law (which knows nothing of transport mean free paths), and the step against both."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

from paper_2203_09467_b200 import workloads as W

ME = 0.51099895
RE = 2.8179403262e-13
HBARC = 197.3269804e-13          # MeV cm


def _law(emo, Z, Am, T):
    """screening parameter A (oracle, pinned in test_oracle_msc.py), cutoff t_m and prefactor of the law, written here"""
    A = emo.lib().emo_msc_screening(Z, T)
    pc2 = T * (T + 2 * ME)
    bpc = pc2 / (T + ME)
    pref = 2 * math.pi * Z * (Z + 1) * (RE * ME / bpc) ** 2
    t_m = min(2.0, 0.5 * HBARC ** 2 / (pc2 * (1.4e-13 * Am ** (1 / 3)) ** 2))
    return A, t_m, pref


def _infinite(material, **phys):
    ph = dict(process_mask=0, msc=2, msc_fr=0.2, msc_smin=1e-3)
    ph.update(phys)
    return dict(name="msc2_pin", seed=12, materials=[material], surfaces=[],
                volumes=[dict(surf=[], sense=[], material=0, tally=0)], field=(0.0, 0.0, 0.0),
                physics=W.physics(**ph), n_slots=1024, queue_capacity=1 << 12)


def _interp(Tab, ph, E):
    n = ph["n_E"]
    t = (math.log(E) - math.log(ph["E_min"])) * (n - 1) / math.log(ph["E_max"] / ph["E_min"])
    j = min(max(int(math.floor(t)), 0), n - 2)
    f = min(max(t - j, 0.0), 1.0)
    return (1 - f) * Tab[j] + f * Tab[j + 1]


@pytest.mark.parametrize("Z,Am", [(6, 12.011), (29, 63.546), (82, 207.2)])
@pytest.mark.parametrize("T", [0.001, 0.01, 0.3, 5.0, 200.0, 2e4])
def test_second_transport_cross_section_is_the_integral_of_the_law(emo, Z, Am, T):
    L = emo.lib()
    A, t_m, pref = _law(emo, Z, Am, T)
    # Int (1 - P_2(mu)) dsigma, 1 - P_2 = (3/2)(1 - mu^2), in y = ln t (the peak at t ~ 2A)
    f = lambda y: pref * 1.5 * math.exp(y) * (2 - math.exp(y)) / (math.exp(y) + 2 * A) ** 2 * math.exp(y)
    val, _ = integrate.quad(f, math.log(2 * A) - 40.0, math.log(t_m), limit=400, epsabs=0, epsrel=1e-12)
    s2 = L.emo_msc_sigma2(Z, Am, T)
    assert s2 == pytest.approx(val, rel=1e-8)
    kappa = s2 / L.emo_msc_sigma1(Z, Am, T)
    assert 1.0 < kappa < 3.0                       # 3 for small angles only, 1 for isotropic scattering
    if A < 1e-6 * t_m:                             # small angles: 1 - P_2 -> 3 (1 - mu) up to the non-logarithmic term
        assert kappa > 2.6


def test_lewis_moments_in_extended_precision(emo):
    """The oracle's conditioned forms against Lewis' formulas as printed, in 50 digits, from tau = 1e-9 (where the
    printed form of <x^2 + y^2> cancels to 27 digits) to complete diffusion, kappa from nearly isotropic to 3."""
    L = emo.lib()
    mp.mp.dps = 60
    for x in (1e-12, 1e-5, 0.01, 0.3, 0.4999, 0.5, 0.77, 3.0, 40.0, 700.0):
        xm = mp.mpf(x)
        ref = (xm * xm / 2 - xm + 1 - mp.exp(-xm)) / xm ** 3
        assert L.emo_msc_phi3(x) == pytest.approx(float(ref), rel=4e-15)
    lam1 = 0.37
    for tau in (1e-9, 1e-6, 1e-3, 0.05, 0.2, 1.0, 6.0, 90.0):
        t = tau * lam1
        z = mp.mpf(lam1) * (1 - mp.exp(-mp.mpf(t) / mp.mpf(lam1)))
        assert L.emo_msc_geom_length(t, 1 / lam1) == pytest.approx(float(z), rel=1e-14)
        for kappa in (1.004, 1.3, 2.0, 2.71, 3.0):
            il1, il2 = 1 / lam1, kappa / lam1
            tm, km = mp.mpf(t) * mp.mpf(il1), mp.mpf(il2) / mp.mpf(il1)
            br = tm - (km + 1) / km + km / (km - 1) * mp.exp(-tm) - mp.exp(-km * tm) / (km * (km - 1))
            ref = 4 / (3 * mp.mpf(il1) ** 2) * br
            # conditioning of either form: the difference of two terms that agree to (kappa - 1)
            assert L.emo_msc_lateral_r2(t, il1, il2) == pytest.approx(float(ref), rel=1e-13 + 2e-15 / (kappa - 1))
    # small-path limits: z -> t (1 - tau / 2), <r^2> -> (2/9) kappa t^3 / lambda_1 (Fermi's (2/3) t^3 / lambda_1 at kappa = 3)
    assert L.emo_msc_lateral_r2(1e-6, 2.0, 6.0) == pytest.approx(2 / 9 * 3 * 1e-18 * 2.0, rel=1e-5)
    assert L.emo_msc_geom_length(0.0, 5.0) == 0.0 and L.emo_msc_lateral_r2(0.0, 5.0, 9.0) == 0.0
    assert L.emo_msc_geom_length(2.0, 0.0) == 2.0          # no scattering: the geometric path is the true path


def test_lewis_moments_by_brute_force_single_scattering(emo):
    """Collision by collision: exponential free paths, polar angles from the screened Rutherford law up to t_m (inverse
    of its distribution function), uniform azimuths, 40 000 electrons of 2 MeV in lead over a true path of
    0.3 lambda_1 (about 460 collisions each).  The mean displacement along the start direction and the mean square
    lateral displacement must be what emo_msc_geom_length / emo_msc_lateral_r2 give for lambda_1, lambda_2 from
    emo_msc_sigma1 / emo_msc_sigma2 -- the simulation uses neither."""
    L = emo.lib()
    Z, Am, T = 82, 207.2, 2.0
    A, t_m, pref = _law(emo, Z, Am, T)
    sig_el = pref * t_m / (2 * A * (t_m + 2 * A))            # Int dsigma, in units where the law's prefactor is `pref`
    s1, s2 = L.emo_msc_sigma1(Z, Am, T), L.emo_msc_sigma2(Z, Am, T)
    il1, il2 = s1 / sig_el, s2 / sig_el                     # 1/lambda_1, 1/lambda_2 in units of the elastic mean free path
    tau = 0.3
    t_tot = tau / il1
    assert 300 < t_tot < 700
    rng = np.random.default_rng(2024)
    n = 40000
    x = np.zeros((n, 3))
    u = np.tile(np.array([0.0, 0.0, 1.0]), (n, 1))
    left = np.full(n, t_tot)
    while True:
        act = left > 0
        if not act.any():
            break
        step = np.minimum(rng.exponential(1.0, n), left) * act
        x += step[:, None] * u
        left = left - step
        xi = rng.random(n) * t_m / (t_m + 2 * A)
        tc = 2 * A * xi / (1 - xi)                           # 1 - cos(theta) of this collision
        st = np.sqrt(tc * (2 - tc))
        phi = 2 * math.pi * rng.random(n)
        # rotate u by (theta, phi): frame e1, e2 perpendicular to u
        a = np.where(np.abs(u[:, 2:3]) < 0.9, np.array([[0.0, 0.0, 1.0]]), np.array([[1.0, 0.0, 0.0]]))
        e1 = np.cross(u, a)
        e1 /= np.linalg.norm(e1, axis=1, keepdims=True)
        e2 = np.cross(u, e1)
        un = (1 - tc)[:, None] * u + (st * np.cos(phi))[:, None] * e1 + (st * np.sin(phi))[:, None] * e2
        u = np.where((left > 0)[:, None], un / np.linalg.norm(un, axis=1, keepdims=True), u)
    z, r2 = x[:, 2], x[:, 0] ** 2 + x[:, 1] ** 2
    want_z = L.emo_msc_geom_length(t_tot, il1)
    want_r2 = L.emo_msc_lateral_r2(t_tot, il1, il2)
    assert abs(z.mean() - want_z) < 4 * z.std() / math.sqrt(n)
    assert abs(r2.mean() - want_r2) < 4 * r2.std() / math.sqrt(n)
    assert want_z < 0.9 * t_tot and want_r2 > 0.01 * t_tot ** 2           # both corrections are far from nothing here
    assert abs(u[:, 2].mean() - math.exp(-tau)) < 4 * u[:, 2].std() / math.sqrt(n)     # and Lewis' <cos>


def test_second_table_is_the_sum_over_the_elements_and_off_without_the_option(emo):
    desc = _infinite(W.PBWO4)
    P = emo.Problem(desc)
    ph = desc["physics"]
    n = ph["n_E"]
    E = np.exp(np.log(ph["E_min"]) + np.arange(n) * np.log(ph["E_max"] / ph["E_min"]) / (n - 1))
    tab, m, L = P.table(0, "msc2"), W.PBWO4, emo.lib()
    for j in (0, 31, 128, n - 1):
        ref = sum(m["rho"] * 6.02214076e23 * w / A * L.emo_msc_sigma2(Z, A, float(E[j]))
                  for Z, A, w in zip(m["Z"], m["A"], m["w"]))
        assert tab[j] == pytest.approx(ref, rel=1e-13)
    assert np.all(tab > P.table(0, "msc"))                  # lambda_2 < lambda_1 at every energy
    assert np.all(emo.Problem(_infinite(W.PBWO4, msc=1)).table(0, "msc2") == 0.0)


def _tracks(emo, n, E, pt, x=(0.0, 0.0, 0.0), u=(0.6, 0.0, 0.8), vol=0):
    trk = (emo.Track * n)()
    for i in range(n):
        trk[i].x[:] = list(x)
        trk[i].u[:] = list(u)
        trk[i].E, trk[i].tid, trk[i].prim, trk[i].step = E, 1000 + i, 3, 4
        trk[i].vol, trk[i].surf, trk[i].ptype, trk[i].alive = vol, -1, pt, 1
    return trk


@pytest.mark.parametrize("pt,E", [(1, 0.2), (1, 3.0), (2, 40.0), (1, 900.0)])
def test_step_moves_by_the_geometric_length_and_spreads_by_lewis(emo, pt, E):
    """One step of 6000 tracks in the same state (different histories) in unbounded lead: every track has the true path
    t of the step limit, lies EXACTLY z(t) ahead of its start along the old direction (the displacement is
    perpendicular to it), loses the energy of the true path, and the mean square of the sideways shift is Lewis'."""
    desc = _infinite(W.PB)
    ph = desc["physics"]
    P = emo.Problem(desc)
    L = emo.lib()
    iL1, iL2 = P.table(0, "msc"), P.table(0, "msc2")
    Rt, Dt = P.table(0, "range_em" if pt == 1 else "range_ep"), P.table(0, "dedx_em" if pt == 1 else "dedx_ep")
    n = 6000
    u0 = np.array([0.6, 0.0, 0.8])
    res = P.step_batch(_tracks(emo, n, E, pt), 12)
    R, lam = _interp(Rt, ph, E), 1 / _interp(iL1, ph, E)
    t_true = min(max(ph["msc_fr"] * max(R, lam), ph["msc_smin"]),
                 R if R <= ph["rho_R"] else ph["alpha_R"] * R + ph["rho_R"] * (1 - ph["alpha_R"]) * (2 - ph["rho_R"] / R))
    z = L.emo_msc_geom_length(t_true, 1 / lam)
    assert z < t_true
    lat2 = np.empty(n)
    for i in range(n):
        r = res[i]
        xx = np.array(r.trk.x[:])
        assert r.s == pytest.approx(t_true, rel=1e-13) and r.n_draws == 3      # interaction length + the two of the deflection
        assert xx @ u0 == pytest.approx(z, rel=1e-12)
        lat2[i] = xx @ xx - (xx @ u0) ** 2
    E1 = res[0].trk.E
    dE = t_true * _interp(Dt, ph, E)
    if dE <= ph["lin_loss"] * E:
        assert E - E1 == pytest.approx(dE, rel=1e-12)                   # the loss of the TRUE path
    tau = 0.5 * (1 / lam + _interp(iL1, ph, E1)) * t_true
    assert res[0].msc_tau == pytest.approx(tau, rel=1e-13)
    want = L.emo_msc_lateral_r2(t_true, 0.5 * (1 / lam + _interp(iL1, ph, E1)), 0.5 * (_interp(iL2, ph, E) + _interp(iL2, ph, E1)))
    assert abs(lat2.mean() - want) < 4 * lat2.std() / math.sqrt(n), (lat2.mean(), want)
    # the shift points along the transverse part of the new direction
    r = res[7]
    xx, u1 = np.array(r.trk.x[:]), np.array(r.trk.u[:])
    shift = xx - (xx @ u0) * u0
    perp = u1 - (u1 @ u0) * u0
    assert np.linalg.norm(np.cross(shift, perp)) < 1e-12 * np.linalg.norm(shift) * np.linalg.norm(perp) + 1e-300
    assert shift @ perp > 0


def test_boundary_cut_step_and_displacement_inside_the_cell(emo):
    """A lead slab 0 < z < 2 um between two thicker ones, e- of 3 MeV.  (a) Heading for the far face: the step ends ON
    it after the geometric length g = 2 um, stands for the true path t g / z(t), and is not displaced.  (b) Travelling
    along the slab from its middle: the sideways shift (tens of um unclipped) stops at 0.9 of the distance to the face
    it points at; the track is still in its cell."""
    thick = 2e-4
    surfaces = [(W.PZ, -1.0), (W.PZ, 0.0), (W.PZ, thick), (W.PZ, 1.0)]
    volumes = [dict(surf=[k, k + 1], sense=[1, -1], material=0, tally=k) for k in range(3)]
    desc = dict(name="msc2_slab", seed=12, materials=[W.PB], surfaces=surfaces, volumes=volumes, field=(0.0, 0.0, 0.0),
                physics=W.physics(process_mask=0, msc=2, msc_fr=0.2, msc_smin=1e-3), n_slots=1024, queue_capacity=1 << 12)
    ph = desc["physics"]
    P = emo.Problem(desc)
    L = emo.lib()
    E = 3.0
    lam = 1 / _interp(P.table(0, "msc"), ph, E)
    R = _interp(P.table(0, "range_em"), ph, E)
    t_lim = max(ph["msc_fr"] * max(R, lam), ph["msc_smin"])
    z_lim = L.emo_msc_geom_length(t_lim, 1 / lam)
    assert z_lim > 10 * thick
    # (a)
    trk = _tracks(emo, 50, E, 1, x=(0.0, 0.0, 0.0), u=(0.0, 0.0, 1.0), vol=1)
    for i in range(50):
        trk[i].surf = 1
    for r in P.step_batch(trk, 12):
        assert r.action == 3 and r.trk.surf == 2 and r.trk.vol == 2
        assert r.s == pytest.approx(t_lim * thick / z_lim, rel=1e-13)
        assert r.trk.x[2] == pytest.approx(thick, rel=1e-15) and r.trk.x[0] == 0.0 and r.trk.x[1] == 0.0
    # (b)
    n = 400
    res = P.step_batch(_tracks(emo, n, E, 1, x=(0.0, 0.0, 0.5 * thick), u=(1.0, 0.0, 0.0), vol=1), 12)
    clipped = 0
    for r in res:
        xx = np.array(r.trk.x[:])
        assert r.action == 5 and r.trk.vol == 1 and 0.0 < xx[2] < thick and P.locate(xx) == 1
        assert xx[0] == pytest.approx(z_lim, rel=1e-13)                  # the move along the old direction
        u1 = np.array(r.trk.u[:])
        perp = u1 - u1[0] * np.array([1.0, 0, 0])
        dh = perp / np.linalg.norm(perp)
        if abs(dh[2]) > 0.2:
            reach = 0.9 * (0.5 * thick) / abs(dh[2])                     # 0.9 x the distance to the face along the shift
            shift = np.linalg.norm(xx - np.array([z_lim, 0.0, 0.5 * thick]))
            if shift == pytest.approx(reach, rel=1e-9):
                clipped += 1
            else:
                assert shift < reach
    assert clipped > n // 4


def test_shower_with_the_spatial_moments_closes_energy_and_is_reproducible(emo):
    desc, prim = W.config2(6)
    desc = dict(desc, physics=dict(desc["physics"], msc=2, fluct=1))
    P = emo.Problem(desc)
    a = P.transport(prim, 5, n_threads=1, per_primary=True)
    b = P.transport(prim, 5, n_threads=4, per_primary=True)
    assert np.array_equal(a["per_prim"], b["per_prim"])
    assert a["edep"].sum() + a["escaped"] + a["looper"] == pytest.approx(a["E_in"], rel=1e-9)
    c = emo.Problem(dict(desc, physics=dict(desc["physics"], msc=1))).transport(prim, 5)
    assert c["steps"][1] != a["steps"][1]                    # the option changes the histories


def test_lateral_shower_containment_in_moliere_radii(emo):
    """What multiple scattering is FOR in a shower, pinned by the PDG review ("Passage of particles through matter",
    electromagnetic cascades): the transverse size scales with the Moliere radius R_M = X0 (21.2 MeV / E_c); on
    average 10 % of the energy lies outside a cylinder of radius R_M, about 1 % outside 3.5 R_M.  200 showers of 1 GeV
    in lead rings of R_M / 4 around the beam axis, 40 X0 deep.  With the deflection and the spatial moments on: 88 / 95 /
    99 % inside 1 / 2 / 3.5 R_M; with multiple scattering off the shower is far too narrow (97 % inside 1 R_M), so the
    pin does see the model."""
    X0 = emo.Problem(W.config1(1)[0]).material_info(0)["X0"]
    RM = X0 * 21.2 / (610.0 / (82 + 1.24))
    assert RM == pytest.approx(1.62, abs=0.01)                         # cm
    radii = [(k + 1) * 0.25 * RM for k in range(20)] + [60.0]
    surfaces = [(W.PZ, 0.0), (W.PZ, 40 * X0)] + [(W.CZ, r) for r in radii]
    volumes = [dict(surf=[0, 1, 2], sense=[1, -1, -1], material=0, tally=0)]
    volumes += [dict(surf=[0, 1, 1 + k, 2 + k], sense=[1, -1, 1, -1], material=0, tally=k) for k in range(1, len(radii))]
    inside = {}
    for msc in (0, 2):
        desc = dict(name="pb_rings", seed=13, materials=[W.PB], surfaces=surfaces, volumes=volumes, field=(0.0, 0.0, 0.0),
                    physics=W.physics(msc=msc), n_slots=1 << 16, queue_capacity=1 << 20)
        r = emo.Problem(desc).transport(W._prim(200, 1, 1000.0, (0, 0, 0), (0, 0, 1), 0, 0), 13)
        assert r["edep"].sum() + r["escaped"] + r["looper"] == pytest.approx(r["E_in"], rel=1e-9)
        cum = np.cumsum(r["edep"]) / r["edep"].sum()
        inside[msc] = (float(cum[3]), float(cum[7]), float(cum[13]))     # 1, 2, 3.5 R_M
    assert 0.85 < inside[2][0] < 0.93 and 0.93 < inside[2][1] < 0.975 and inside[2][2] > 0.975, inside
    assert inside[0][0] > 0.95, inside
