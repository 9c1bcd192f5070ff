"""Pins for the oracle's energy-loss fluctuations of e+- (DESIGN.md R-FLUCT): the variance per unit
path against a quadrature of W^2 times the pinned Moller / Bhabha laws and against Bohr's leading term, the sampler
against the normal law it is built on and its bounds, one step against a problem without fluctuations, and the
variance of the summed loss over several steps."""
import math

import numpy as np
import pytest
from scipy import integrate, stats

from paper_2203_09467_b200 import workloads as W
from test_oracle_msc import _infinite, _interp

ME = 0.51099895
RE = 2.8179403262e-13


@pytest.mark.parametrize("pt", [1, 2])
@pytest.mark.parametrize("T,Tcut", [(0.05, 0.01), (1.0, 0.35), (1.0, 0.9), (30.0, 1.0), (3e3, 1.02), (8e4, 0.1)])
def test_second_moment_is_the_integral_of_W2_times_the_law(emo, pt, T, Tcut):
    L = emo.lib()
    dcs = L.emo_moller_dcs if pt == 1 else L.emo_bhabha_dcs
    x = min(Tcut / T, 0.5 if pt == 1 else 1.0)
    val, _ = integrate.quad(lambda e: (e * T) ** 2 * dcs(T, e), 0.0, x, epsabs=0, epsrel=1e-12, limit=200)
    assert L.emo_loss_second_moment(pt, T, Tcut) == pytest.approx(val, rel=1e-9)


def test_second_moment_tends_to_bohrs_value(emo):
    """Transfers far below the kinetic energy follow the Rutherford law: Int W^2 dsigma -> 2 pi re^2 me Tup / beta^2."""
    L = emo.lib()
    for pt in (1, 2):
        for T in (0.1, 10.0, 1e4):
            g = T / ME + 1
            b2 = 1 - 1 / g ** 2
            for x, tol in ((1e-3, 5e-3), (1e-5, 5e-5)):
                bohr = 2 * math.pi * RE ** 2 * ME * (x * T) / b2
                assert L.emo_loss_second_moment(pt, T, x * T) == pytest.approx(bohr, rel=tol)


def test_sampler_is_normal_about_the_mean_and_stays_inside_its_bounds(emo):
    L = emo.lib()
    rng = np.random.default_rng(2)
    u = rng.random((60000, 2))
    # sigma << mean: never clamped
    dE, V, E = 2.0, 0.09, 100.0
    d = np.array([L.emo_fluctuate_loss(dE, V, E, a, b) for a, b in u])
    assert abs(d.mean() - dE) < 4.5 * d.std() / math.sqrt(len(d))
    assert d.var() == pytest.approx(V, rel=0.03)
    assert stats.kstest((d - dE) / math.sqrt(V), "norm").pvalue > 1e-3
    # the same uniforms give the same normal deviate: linear in sqrt(V)
    z = (d - dE) / 0.3
    d2 = np.array([L.emo_fluctuate_loss(dE, 4 * V, E, a, b) for a, b in u[:2000]])
    inside = np.abs(z[:2000]) < 3.3                                  # beyond, 2 dE bounds it
    assert np.allclose(d2[inside], dE + 0.6 * z[:2000][inside], rtol=0, atol=1e-12) and inside.sum() > 1900
    # Box-Muller on the two uniforms, first one radial
    assert L.emo_fluctuate_loss(dE, V, E, 0.5, 0.25) == pytest.approx(dE, abs=1e-15)            # cos(pi/2) = 0
    assert L.emo_fluctuate_loss(dE, V, E, math.exp(-2.0), 0.0) == pytest.approx(dE + 0.3 * 2.0, rel=1e-14)
    assert L.emo_fluctuate_loss(dE, V, E, math.exp(-2.0), 0.5) == pytest.approx(dE - 0.3 * 2.0, rel=1e-14)
    # sigma >> mean: clamped to [0, 2 dE], symmetric, so the mean survives
    d = np.array([L.emo_fluctuate_loss(dE, 25.0, E, a, b) for a, b in u])
    assert d.min() == 0.0 and d.max() == 2 * dE
    assert abs(d.mean() - dE) < 4.5 * d.std() / math.sqrt(len(d))
    # never more than the particle has
    d = np.array([L.emo_fluctuate_loss(dE, 25.0, 3.0, a, b) for a, b in u[:5000]])
    assert d.max() == 3.0 and d.min() == 0.0


@pytest.mark.parametrize("pt", [1, 2])
@pytest.mark.parametrize("msc", [0, 1])
def test_one_step_with_fluctuations_against_the_step_without(emo, pt, msc):
    ph = _infinite(W.SI, msc=msc)["physics"]
    P0 = emo.Problem(_infinite(W.SI, msc=msc, fluct=0))
    P1 = emo.Problem(_infinite(W.SI, msc=msc, fluct=1))
    var = P1.table(0, "var_em" if pt == 1 else "var_ep")
    assert np.all(var > 0) and np.all(P0.table(0, "var_em") == 0)
    L = emo.lib()
    n_fluct = 0
    for k, E in enumerate([0.02, 0.3, 2.0, 25.0, 400.0, 7000.0]):
        trk = (emo.Track * 1)()
        trk[0].x[:] = [0.0, 0.0, 0.0]
        trk[0].u[:] = [0.0, 0.6, 0.8]
        trk[0].E, trk[0].tid, trk[0].prim, trk[0].step = E, 5 + k, 2, 1
        trk[0].vol, trk[0].surf, trk[0].ptype, trk[0].alive = 0, -1, pt, 1
        r0, r1 = P0.step_batch(trk, 31)[0], P1.step_batch(trk, 31)[0]
        assert r1.action == r0.action and r1.s == r0.s                       # the limits do not know about it
        if r0.action == 2 and not r0.trk.alive:                              # range stop: everything is lost
            assert r1.edep == r0.edep
            continue
        x1, x2 = L.emo_draw(31, 2, 5 + k, 1, 1), L.emo_draw(31, 2, 5 + k, 1, 2)     # draws 1 and 2 of the step
        V = r0.s * _interp(var, ph, E)
        want = L.emo_fluctuate_loss(r0.edep, V, E, x1, x2)
        if r1.trk.alive:
            assert r1.edep == pytest.approx(want, rel=1e-13)
            assert r1.trk.E == pytest.approx(E - want, rel=1e-13, abs=1e-13 * E)
            assert r1.n_draws == r0.n_draws + 2 == 3 + 2 * msc
            n_fluct += r1.edep != r0.edep
    assert n_fluct >= 3


def test_variance_of_the_summed_loss_is_the_sum_of_the_step_variances(emo):
    """Six slabs of 0.5 mm Si crossed along z without discrete processes and without multiple scattering: every
    history takes the same six boundary-limited steps, so the summed loss spreads with the variance
    sum_i s Omega^2(E_i) (independent steps, unclamped regime; the E_i differ by a few per cent between histories)."""
    n_layer, d = 7, 0.05
    desc = _infinite(W.SI, msc=0, fluct=1)
    desc.update(surfaces=[(W.PZ, k * d) for k in range(n_layer + 1)],
                volumes=[dict(surf=[k, k + 1], sense=[1, -1], material=0, tally=0) for k in range(n_layer)])
    ph = desc["physics"]
    P = emo.Problem(desc)
    var, D = P.table(0, "var_em"), P.table(0, "dedx_em")
    n, k_steps, E0 = 5000, 6, 3.0
    trk = (emo.Track * n)()
    for i in range(n):
        trk[i].x[:] = [0.0, 0.0, 0.0]
        trk[i].u[:] = [0.0, 0.0, 1.0]
        trk[i].E, trk[i].tid, trk[i].prim, trk[i].step = E0, 1, i, 0
        trk[i].vol, trk[i].surf, trk[i].ptype, trk[i].alive = 0, 0, 1, 1
    V, mean_loss, E = 0.0, 0.0, E0
    for _ in range(k_steps):
        V += d * _interp(var, ph, E)                      # along the mean history
        mean_loss += d * _interp(D, ph, E)
        E = E0 - mean_loss
        out = P.step_batch(trk, 41)
        assert all(o.action == 3 and abs(o.s - d) < 1e-12 for o in out)
        for i in range(n):
            trk[i] = out[i].trk
    loss = E0 - np.array([t.E for t in trk])
    assert 3.0 * math.sqrt(V / k_steps) < mean_loss / k_steps          # the bounds sit beyond 3 sigma of a step: ~1 % of the variance
    assert loss.mean() == pytest.approx(mean_loss, rel=1e-2)
    assert loss.var() == pytest.approx(V, rel=0.08)


def test_shower_with_fluctuations_closes_energy(emo):
    desc, prim = W.get(1, 40)
    desc = dict(desc, physics=dict(desc["physics"], fluct=1))
    o = emo.Problem(desc).transport(prim, desc["seed"], per_primary=True)
    pp = o["per_prim"]
    assert np.all(np.abs(pp[:, 0] + pp[:, 1] + pp[:, 2] - pp[:, 4]) <= 1e-9 * pp[:, 4])
