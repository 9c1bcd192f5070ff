"""Pins for the oracle's discrete interactors: each sampler's histogram against
quadrature of the differential cross section, plus the conservation laws / closed-form kinematics."""
import math

import numpy as np
import pytest
from scipy.integrate import quad

ME, RE = 0.51099895, 2.8179403262e-13
N = 40000


def _chi2(samples, pdf, lo, hi, nbins=24):
    edges = np.linspace(lo, hi, nbins + 1)
    h, _ = np.histogram(samples, bins=edges)
    p = np.array([quad(pdf, edges[i], edges[i + 1], epsrel=1e-9)[0] for i in range(nbins)])
    p /= p.sum()
    exp = p * len(samples)
    keep = exp > 5
    return (((h - exp) ** 2 / np.where(keep, exp, 1))[keep]).sum() / max(keep.sum() - 1, 1)


def _unit(v):
    return np.linalg.norm(v, axis=1)


U = np.array([0.36, -0.48, 0.8])


@pytest.mark.parametrize("E", [0.01, 0.5, 10.0, 1000.0])
def test_compton_sampler(emo, E):
    r = emo.sample("compton", N, u=U, E=E)
    E1, Te, ug, ue = r["a"], r["b"], r["v1"], r["v2"]
    k = E / ME
    mu = ug @ U
    # closed-form kinematics: E' = E / (1 + kappa (1 - mu)); energy and momentum closure
    assert np.allclose(E1, E / (1 + k * (1 - mu)), rtol=1e-12)
    assert np.allclose(E1 + Te, E, rtol=1e-15)
    pe = np.sqrt(Te * (Te + 2 * ME))
    clos = E * U[None, :] - E1[:, None] * ug - pe[:, None] * ue
    assert np.abs(clos).max() < 1e-11 * E
    assert np.allclose(_unit(ug), 1, atol=1e-14) and np.allclose(_unit(ue), 1, atol=1e-14)
    eps = E1 / E
    e0 = 1 / (1 + 2 * k)
    assert eps.min() >= e0 * (1 - 1e-12) and eps.max() <= 1

    def pdf(e):     # Klein-Nishina in eps: (1/eps + eps)(1 - eps sin^2 / (1 + eps^2))
        t = (1 - e) / (k * e)
        return (1 / e + e) * (1 - e * t * (2 - t) / (1 + e * e))
    assert _chi2(eps, pdf, e0, 1.0) < 1.8
    # azimuth is uniform
    perp = ug - mu[:, None] * U[None, :]
    a = np.array([0.8, 0.6, 0.0])
    b = np.cross(U, a)
    phi = np.arctan2(perp @ b, perp @ a)
    assert _chi2(phi, lambda x: 1.0, -math.pi, math.pi, 12) < 2.2


@pytest.mark.parametrize("E", [0.001, 0.1, 1.0])
def test_photoelectron_angle(emo, E):
    r = emo.sample("photo", N, u=U, E=E)
    mu = r["v1"] @ U
    g = E / ME + 1; b = math.sqrt(1 - 1 / g ** 2)
    assert _chi2(mu, lambda m: (1 - m * m) / (1 - b * m) ** 4, -1, 1) < 1.8
    # rejection efficiency is 2/3 at every energy: 2 draws per trial + 1 azimuth
    trials = (r["n_draws"] - 1) / 2
    assert 1 / trials.mean() == pytest.approx(2 / 3, abs=0.01)
    want = {0.001: 0.050, 0.1: 0.460, 1.0: 0.9005}[E]
    assert mu.mean() == pytest.approx(want, abs=0.01)


@pytest.mark.parametrize("Z,E", [(82, 3.0), (82, 30.0), (82, 1000.0), (18, 100.0)])
def test_pair_sampler(emo, Z, E):
    L = emo.lib()
    r = emo.sample("pair", N, u=U, Z=Z, E=E)
    assert r["ok"].all()
    Tm, Tp = r["a"], r["b"]
    assert np.allclose(Tm + Tp + 2 * ME, E, rtol=1e-14)             # energy pin
    assert Tm.min() >= 0 and Tp.min() >= 0
    eps = (Tm + ME) / E
    assert _chi2(eps, lambda e: L.emo_pair_dcs(Z, E, e), ME / E, 1 - ME / E, 30) < 1.8
    # which lepton takes eps is a fair coin
    assert abs((eps < 0.5).mean() - 0.5) < 0.01
    # leptons are emitted back to back in azimuth and forward-peaked (~1/gamma)
    um, up = r["v1"], r["v2"]
    pm = um - (um @ U)[:, None] * U; pp = up - (up @ U)[:, None] * U
    cosd = (pm * pp).sum(1) / (np.linalg.norm(pm, axis=1) * np.linalg.norm(pp, axis=1))
    assert np.allclose(cosd, -1, atol=1e-6)
    assert np.allclose(_unit(um), 1, atol=1e-14)


def test_pair_null_below_screening_limit(emo):
    r = emo.sample("pair", 50, u=U, Z=82, E=1.2)       # dmin >= dmax: no phase space in this model
    assert not r["ok"].any() and (r["n_draws"] == 0).all()


def test_boosted_isotropic_angle_is_exact_inverse_cdf(emo):
    # brems photon polar angle: p(mu) ~ (1 - beta mu)^-2
    T = 2.0
    r = emo.sample("brems", N, u=U, T=T, kc=0.1)
    b = math.sqrt(T * (T + 2 * ME)) / (T + ME)
    mu = r["v1"] @ U
    assert _chi2(mu, lambda m: (1 - b * m) ** -2, -1, 1, 30) < 1.8


@pytest.mark.parametrize("T", [5.0, 1e3, 1e5])
def test_emission_angle_keeps_its_precision_at_high_energy(emo, T):
    """The emission angles of bremsstrahlung photons are ~1/gamma.  The sampler forms t = 1 - mu directly
    (DESIGN.md section 6), so the ANGLE must agree with a 50-digit evaluation of the inverse distribution function
    mu = (v + beta) / (beta v + 1), v = 2 xi - 1 (SURVEY C6 "Common"), to 1e-13 relative at every energy -- a
    rounded mu would lose gamma^2 = 4e10 of that at 100 GeV -- and so must the recoil direction, which is fixed by
    p u = k u_gamma + p' u'."""
    import mpmath as mp
    mp.mp.dps = 50
    n = 200
    Z = np.array([0.0, 0.0, 1.0])                                  # incident direction: angles are read off x, y
    r = emo.sample("brems", n, u=Z, T=T, kc=0.02)
    L = emo.lib()
    worst = worst_recoil = 0.0
    for i in range(n):
        nd = int(r["n_draws"][i])
        xi = mp.mpf(L.emo_draw(12345, i, 7, 3, nd - 2))           # the polar draw: last but one of the sampler
        Tm, me = mp.mpf(T), mp.mpf(ME)
        beta = mp.sqrt(Tm * (Tm + 2 * me)) / (Tm + me)
        v = 2 * xi - 1
        one_minus_mu = (1 - beta) * (1 - v) / (1 + beta * v)
        sin_ref = mp.sqrt(one_minus_mu * (2 - one_minus_mu))
        ug = r["v1"][i]
        sin_got = math.hypot(ug[0], ug[1])
        worst = max(worst, abs(sin_got - float(sin_ref)) / float(sin_ref))
        # recoil: transverse momentum balance p' sin' = k sin, longitudinal p' cos' = p - k mu
        k = mp.mpf(float(r["a"][i]))
        p = mp.sqrt(Tm * (Tm + 2 * me))
        px, pz = -k * sin_ref, p - k * (1 - one_minus_mu)
        sin1_ref = abs(px) / mp.sqrt(px * px + pz * pz)
        u1 = r["v2"][i]
        worst_recoil = max(worst_recoil, abs(math.hypot(u1[0], u1[1]) - float(sin1_ref)) / float(sin1_ref))
    assert worst < 1e-13 and worst_recoil < 1e-13, (worst, worst_recoil)


@pytest.mark.parametrize("T,kc", [(1.0, 0.1), (100.0, 0.175), (1e4, 0.0183)])
def test_brems_sampler(emo, T, kc):
    r = emo.sample("brems", N, u=U, T=T, kc=kc)
    assert r["ok"].all()
    k, T1, ug, u1 = r["a"], r["b"], r["v1"], r["v2"]
    assert np.allclose(k + T1, T, rtol=1e-14) and k.min() >= kc * (1 - 1e-12) and k.max() <= T
    assert _chi2(np.log(k), lambda lk: 4 / 3 - 4 * (math.exp(lk) / T) / 3 + (math.exp(lk) / T) ** 2,
                 math.log(kc), math.log(T)) < 1.8
    p = math.sqrt(T * (T + 2 * ME))
    q = p * U[None, :] - k[:, None] * ug
    assert np.allclose(u1, q / np.linalg.norm(q, axis=1)[:, None], atol=1e-12)
    assert not emo.sample("brems", 5, u=U, T=kc * 0.99, kc=kc)["ok"].any()


@pytest.mark.parametrize("kind,T,Tcut", [("moller", 3.0, 1.0), ("moller", 100.0, 1.0), ("moller", 1e4, 0.35),
                                          ("bhabha", 3.0, 1.0), ("bhabha", 100.0, 1.0), ("bhabha", 0.05, 0.01)])
def test_ionisation_samplers(emo, kind, T, Tcut):
    L = emo.lib()
    r = emo.sample(kind, N, u=U, T=T, Tcut=Tcut)
    assert r["ok"].all()
    Td, T1, ud, u1 = r["a"], r["b"], r["v1"], r["v2"]
    emax = 0.5 if kind == "moller" else 1.0
    eps = Td / T
    assert eps.min() >= Tcut / T * (1 - 1e-12) and eps.max() <= emax
    dcs = L.emo_moller_dcs if kind == "moller" else L.emo_bhabha_dcs
    # compare in 1/eps, where the distribution is nearly flat
    assert _chi2(1 / eps, lambda y: dcs(T, 1 / y) / (y * y), 1 / emax, T / Tcut) < 1.8
    # exact two-body kinematics on a free electron at rest: energy and 3-momentum conservation
    assert np.allclose(Td + T1, T, rtol=1e-14)
    p = math.sqrt(T * (T + 2 * ME)); pd = np.sqrt(Td * (Td + 2 * ME)); p1 = np.sqrt(T1 * (T1 + 2 * ME))
    assert np.allclose(ud @ U, Td * (T + 2 * ME) / (p * pd), atol=1e-12)
    clos = p * U[None, :] - pd[:, None] * ud - p1[:, None] * u1
    assert np.abs(clos).max() < 1e-9 * p


def test_ionisation_thresholds(emo):
    assert not emo.sample("moller", 5, u=U, T=2.0, Tcut=1.0)["ok"].any()
    assert not emo.sample("bhabha", 5, u=U, T=1.0, Tcut=1.0)["ok"].any()


@pytest.mark.parametrize("T", [1e-3, 0.1, 1.0, 100.0])
def test_annihilation_in_flight(emo, T):
    r = emo.sample("annih", N, u=U, T=T)
    k1, k2, u1, u2 = r["a"], r["b"], r["v1"], r["v2"]
    g = T / ME + 1
    p = math.sqrt(T * (T + 2 * ME))
    assert np.allclose(k1 + k2, T + 2 * ME, rtol=1e-14)                       # energy
    clos = p * U[None, :] - k1[:, None] * u1 - k2[:, None] * u2               # momentum
    assert np.abs(clos).max() < 1e-10 * (T + 2 * ME)
    eps = k1 / (T + 2 * ME)
    rr = math.sqrt((g - 1) / (g + 1))
    lo, hi = 0.5 * (1 - rr), 0.5 * (1 + rr)
    assert eps.min() >= lo * (1 - 1e-12) and eps.max() <= hi * (1 + 1e-12)
    assert _chi2(eps, lambda e: (1 / e) * (1 + 2 * g / (g + 1) ** 2 - e - 1 / ((g + 1) ** 2 * e)), lo, hi) < 1.8


def test_annihilation_at_rest(emo):
    r = emo.sample("rest", N)
    u1, u2 = r["v1"], r["v2"]
    assert np.array_equal(u1, -u2) and np.allclose(_unit(u1), 1, atol=1e-14)
    assert _chi2(u1[:, 2], lambda m: 1.0, -1, 1, 20) < 1.9
    assert _chi2(np.arctan2(u1[:, 1], u1[:, 0]), lambda m: 1.0, -math.pi, math.pi, 20) < 1.9
    assert (r["n_draws"] == 2).all()


def test_rotation_preserves_polar_angle_and_norm(emo):
    import ctypes as C
    L = emo.lib()
    rng = np.random.default_rng(5)
    dp = C.POINTER(C.c_double)
    for u in (U, np.array([0.0, 0.0, 1.0]), np.array([0.0, 0.0, -1.0]), np.array([1e-16, 0, 1.0])):
        for _ in range(50):
            mu, phi = rng.uniform(-1, 1), rng.uniform(0, 2 * math.pi)
            out = np.zeros(3)
            L.emo_rotate(u.ctypes.data_as(dp), mu, phi, out.ctypes.data_as(dp))
            assert abs(np.linalg.norm(out) - 1) < 1e-14
            assert abs(out @ (u / np.linalg.norm(u)) - mu) < 1e-12
    # phi = 0 and phi = pi/2 are orthogonal displacements of equal size
    a = np.zeros(3); b = np.zeros(3)
    L.emo_rotate(U.ctypes.data_as(dp), 0.3, 0.0, a.ctypes.data_as(dp))
    L.emo_rotate(U.ctypes.data_as(dp), 0.3, math.pi / 2, b.ctypes.data_as(dp))
    pa, pb = a - 0.3 * U, b - 0.3 * U
    assert abs(pa @ pb) < 1e-14 and abs(np.linalg.norm(pa) - np.linalg.norm(pb)) < 1e-14
