"""Pins for the oracle's closed-form cross sections and stopping powers.

Each total cross section is checked against numerical quadrature of the differential cross section
written out here from the textbook formula (a different expression from the closed form under
test), against limits, and against the printed values in tests/golden/.
"""
import math

import numpy as np
import pytest
from scipy.integrate import quad

from conftest import golden

ME, RE, ALPHA, NA = 0.51099895, 2.8179403262e-13, 7.2973525693e-3, 6.02214076e23
BARN = 1e-24


def _pb_problem(emo, Tcut, kcut, **phys):
    from paper_2203_09467_b200 import workloads as W
    m = dict(W.PB); m["Tcut"] = Tcut; m["kcut"] = kcut
    d = dict(materials=[m], surfaces=[], volumes=[dict(surf=[], sense=[], material=0, tally=0)],
             field=(0, 0, 0), physics=W.physics(**phys))
    return emo.Problem(d)


def test_radiation_length_against_pdg_table(emo):
    L = emo.lib()
    for Z, A, x0 in golden("pdg_radiation_length.txt"):
        got = L.emo_X0_elem_gcm2(int(Z), float(A))
        assert got == pytest.approx(float(x0), rel=2e-3), (Z, got)


def test_golden_cross_sections(emo):
    L = emo.lib()
    for kind, a, b, v in golden("cross_sections_barn.txt"):
        a, b, v = float(a), float(b), float(v)
        if kind == "kn":
            assert L.emo_sigma_kn(a) / BARN == pytest.approx(v, rel=1e-12)
        elif kind == "moller":
            assert L.emo_sigma_moller(a, b) / BARN == pytest.approx(v, rel=2e-7)
        elif kind == "bhabha":
            assert L.emo_sigma_bhabha(a, b) / BARN == pytest.approx(v, rel=2e-7)
        elif kind == "annih":
            assert L.emo_sigma_annih(a) / BARN == pytest.approx(v, rel=2e-7)
        elif kind == "pair":
            assert L.emo_sigma_pair(int(a), b) / BARN == pytest.approx(v, rel=5e-4)


def _kn_dcs_dmu(kappa, mu):
    """Klein-Nishina dsigma/dmu per electron (mu = cos theta), textbook form."""
    r = 1.0 / (1.0 + kappa * (1.0 - mu))
    return math.pi * RE * RE * r * r * (r + 1.0 / r - (1.0 - mu * mu))


@pytest.mark.parametrize("E", [1e-3, 5e-3, 0.02, 0.1, 0.511, 2.0, 10.0, 100.0, 1e4])
def test_klein_nishina_total_is_integral_of_dcs(emo, E):
    val, err = quad(lambda mu: _kn_dcs_dmu(E / ME, mu), -1, 1, epsabs=0, epsrel=1e-13, limit=200)
    assert emo.lib().emo_sigma_kn(E) == pytest.approx(val, rel=1e-11)


def test_klein_nishina_thomson_limit(emo):
    sT = 8 * math.pi * RE * RE / 3
    assert sT / BARN == pytest.approx(0.6652458732, rel=1e-9)
    k = 1e-6
    assert emo.lib().emo_sigma_kn(k * ME) == pytest.approx(sT * (1 - 2 * k), rel=1e-10)


def test_photoelectric_scaling(emo):
    L = emo.lib()
    # Z^5 and E^-7/2 scaling, Born K-shell x 5/4 normalisation
    assert L.emo_sigma_pe(82, 1.0) / L.emo_sigma_pe(41, 1.0) == pytest.approx(32.0, rel=1e-13)
    assert L.emo_sigma_pe(82, 0.1) / L.emo_sigma_pe(82, 1.0) == pytest.approx(10 ** 3.5, rel=1e-13)
    sT = 8 * math.pi * RE * RE / 3
    want = 1.25 * 4 * math.sqrt(2) * ALPHA ** 4 * 82 ** 5 * sT * (ME / 1.0) ** 3.5
    assert L.emo_sigma_pe(82, 1.0) == pytest.approx(want, rel=1e-13)
    n_pb = 11.35 * NA / 207.2
    assert n_pb * L.emo_sigma_pe(82, 1.0) == pytest.approx(1.556055e-1, rel=1e-6)


@pytest.mark.parametrize("Z,E", [(82, 3.0), (82, 10.0), (82, 49.0), (82, 51.0), (82, 1e3), (18, 100.0), (8, 10.0)])
def test_pair_gl32_against_adaptive_quadrature(emo, Z, E):
    L = emo.lib()
    e0 = ME / E
    val, _ = quad(lambda e: L.emo_pair_dcs(Z, E, e), e0, 0.5, epsabs=0, epsrel=1e-10, limit=400,
                  points=None)
    assert L.emo_sigma_pair(Z, E) == pytest.approx(2 * val, rel=2e-3)


def test_pair_threshold_symmetry_and_high_energy_limit(emo):
    L = emo.lib()
    assert L.emo_sigma_pair(82, 2 * ME) == 0.0
    assert L.emo_sigma_pair(82, 1.0) == 0.0
    for e in (0.1, 0.3, 0.45):
        assert L.emo_pair_dcs(82, 100.0, e) == pytest.approx(L.emo_pair_dcs(82, 100.0, 1 - e), rel=1e-12)
    # sigma -> (7/9) A / (X0 N_A) (complete screening), within 1 %
    for Z, A in ((82, 207.2), (18, 39.948), (29, 63.546)):
        lim = 7.0 / 9.0 * A / (L.emo_X0_elem_gcm2(Z, A) * NA)
        assert L.emo_sigma_pair(Z, 1e5) == pytest.approx(lim, rel=1.5e-2)


def test_pair_F1_F2_decomposition(emo):
    """DCS bracket = (2/3)(1/2-eps)^2 F1 + (1/3) F2 with F1 = 3phi1-phi2-F, F2 = 1.5phi1+0.5phi2-F."""
    L = emo.lib()
    Z, E = 82, 20.0
    F = 8.0 / 3.0 * math.log(Z)
    fc = L.emo_fc(Z)
    xi = math.log(1440 * Z ** (-2 / 3)) / (math.log(183 * Z ** (-1 / 3)) - fc)
    for eps in (0.1, 0.2, 0.35, 0.49):
        d = 136 * Z ** (-1 / 3) * (ME / E) / (eps * (1 - eps))
        if d <= 1:
            p1 = 20.867 - 3.242 * d + 0.625 * d * d; p2 = 20.209 - 1.930 * d - 0.086 * d * d
        else:
            p1 = p2 = 21.12 - 4.184 * math.log(d + 0.952)
        F1, F2 = 3 * p1 - p2 - F, 1.5 * p1 + 0.5 * p2 - F
        br = (2 / 3) * (0.5 - eps) ** 2 * F1 + F2 / 3
        want = ALPHA * RE * RE * Z * (Z + xi) * br
        assert L.emo_pair_dcs(Z, E, eps) == pytest.approx(want, rel=1e-12)


@pytest.mark.parametrize("T,Tcut", [(3.0, 1.0), (100.0, 1.0), (1e4, 0.35), (0.05, 0.01), (2.5, 1.0)])
def test_moller_bhabha_totals_are_integrals_of_dcs(emo, T, Tcut):
    L = emo.lib()
    x = Tcut / T
    vm, _ = quad(lambda e: L.emo_moller_dcs(T, e), x, 0.5, epsabs=0, epsrel=1e-12, limit=400)
    vb, _ = quad(lambda e: L.emo_bhabha_dcs(T, e), x, 1.0, epsabs=0, epsrel=1e-12, limit=400)
    assert L.emo_sigma_moller(T, Tcut) == pytest.approx(vm, rel=1e-10)
    assert L.emo_sigma_bhabha(T, Tcut) == pytest.approx(vb, rel=1e-10)


def test_moller_bhabha_thresholds_and_rutherford_limit(emo):
    L = emo.lib()
    assert L.emo_sigma_moller(1.9, 1.0) == 0.0 and L.emo_sigma_moller(2.0, 1.0) == 0.0
    assert L.emo_sigma_bhabha(1.0, 1.0) == 0.0
    # soft limit eps -> 0: both reduce to the Rutherford form 2 pi re^2 / (beta^2 (gamma-1) eps^2)
    T, eps = 50.0, 1e-5
    g = T / ME + 1; b2 = 1 - 1 / g ** 2
    ruth = 2 * math.pi * RE * RE / (b2 * (g - 1) * eps * eps)
    assert L.emo_moller_dcs(T, eps) == pytest.approx(ruth, rel=1e-4)
    assert L.emo_bhabha_dcs(T, eps) == pytest.approx(ruth, rel=1e-4)
    # Moller DCS is symmetric under eps <-> 1-eps (identical particles)
    assert L.emo_moller_dcs(T, 0.2) == pytest.approx(L.emo_moller_dcs(T, 0.8), rel=1e-13)


@pytest.mark.parametrize("T", [1e-3, 0.1, 1.0, 100.0, 1e4])
def test_annihilation_total_is_integral_of_heitler_dcs(emo, T):
    g = T / ME + 1
    r = math.sqrt((g - 1) / (g + 1))
    lo, hi = 0.5 * (1 - r), 0.5 * (1 + r)

    def dcs(e):   # Heitler: dsigma/deps, eps = k1 / (T + 2 me)
        return math.pi * RE * RE / (g - 1) / e * (1 + 2 * g / (g + 1) ** 2 - e - 1 / ((g + 1) ** 2 * e))
    val, _ = quad(dcs, lo, hi, epsabs=0, epsrel=1e-12, limit=400)
    assert emo.lib().emo_sigma_annih(T) == pytest.approx(val, rel=1e-9)


def test_bremsstrahlung_closed_forms(emo):
    L = emo.lib()
    X0 = 0.5612
    for T, kc in ((10.0, 0.175), (1e3, 0.175), (0.5, 0.1)):
        val, _ = quad(lambda k: (1 / X0) / k * (4 / 3 - 4 * (k / T) / 3 + (k / T) ** 2), kc, T, epsrel=1e-12)
        assert L.emo_brems_Sigma(T, kc, X0) == pytest.approx(val, rel=1e-10)
        lo, _ = quad(lambda k: (1 / X0) * (4 / 3 - 4 * (k / T) / 3 + (k / T) ** 2), 0, kc, epsrel=1e-12)
        assert L.emo_brems_dedx(T, kc, X0) == pytest.approx(lo, rel=1e-10)
        # definition of X0: unrestricted radiative loss is exactly T/X0
        assert L.emo_brems_dedx(T, -1.0, X0) == pytest.approx(T / X0, rel=1e-15)
        assert L.emo_brems_dedx(T, 2 * T, X0) == pytest.approx(T / X0, rel=1e-15)
    assert L.emo_brems_Sigma(0.1, 0.175, X0) == 0.0


def _density(hwp, I, b2, g):
    return max(0.0, 2 * math.log(hwp * math.sqrt(b2) * g / I) - 1)


@pytest.mark.parametrize("T", [0.01, 0.1, 1.0, 10.0, 1e3])
def test_unrestricted_collision_loss_reduces_to_icru37(emo, T):
    """Restricted Berger-Seltzer formula with tau_up = tau/2 (e-) or tau (e+) equals the ICRU-37 forms."""
    P = _pb_problem(emo, 1e9, 1e9, E_min=T, E_max=2 * T, n_E=2)       # grid node 0 sits exactly at T
    mi = P.material_info(0)
    tau = T / ME; g = tau + 1; b2 = 1 - 1 / g ** 2
    Im = mi["I"] / ME
    lg = math.log(tau * tau * (tau + 2) / (2 * Im * Im))
    dl = _density(mi["hwp"], mi["I"], b2, g)
    pre = 2 * math.pi * RE * RE * ME * mi["n_e"] / b2
    Fm = 1 - b2 + (tau * tau / 8 - (2 * tau + 1) * math.log(2)) / g ** 2
    Fp = 2 * math.log(2) - b2 / 12 * (23 + 14 / (tau + 2) + 10 / (tau + 2) ** 2 + 4 / (tau + 2) ** 3)
    rad = T / mi["X0"]
    assert P.table(0, "dedx_em")[0] - rad == pytest.approx(pre * (lg + Fm - dl), rel=1e-11)
    assert P.table(0, "dedx_ep")[0] - rad == pytest.approx(pre * (lg + Fp - dl), rel=1e-11)


def _one_material(emo, mat, T, **over):
    """problem of one material whose energy grid starts exactly at T, no production threshold below T"""
    from paper_2203_09467_b200 import workloads as W
    m = dict(mat, Tcut=1e9, kcut=1e9, **over)
    d = dict(materials=[m], surfaces=[], volumes=[dict(surf=[], sense=[], material=0, tally=0)],
             field=(0, 0, 0), physics=W.physics(E_min=T, E_max=2 * T, n_E=2))
    return emo.Problem(d)


def test_printed_collision_stopping_powers(emo):
    """SURVEY C5.8 pin (iii): the printed unrestricted (dE/dx)_col / rho, density effect zero (golden file)."""
    from paper_2203_09467_b200 import workloads as W
    mats = {"Pb": W.PB, "lAr": W.LAR, "Si": W.SI}
    rows = golden("dedx_collision_unrestricted.txt")
    assert len(rows) == 5
    for name, I_eV, T, want in rows:
        T = float(T)
        assert mats[name]["I_eV"] == float(I_eV)
        P = _one_material(emo, mats[name], T)
        mi = P.material_info(0)
        got = (P.table(0, "dedx_em")[0] - T / mi["X0"]) / mi["rho"]
        assert abs(got - float(want)) < 0.6e-4, (name, T, got)          # every printed digit


def test_density_effect_gives_the_fermi_plateau(emo):
    """Density effect (R23), pinned by what it is FOR: once it is on, the collision loss no longer depends
    on the mean excitation energy I (Fermi plateau: only the electron density enters, through the plasma energy),
    and it switches on where hbar omega_p beta gamma = sqrt(e) I.  Below the onset two values of I differ by the
    Bethe logarithm, 2 ln(I_a / I_b) times the prefactor.  A wrong coefficient of the logarithm of delta, a
    missing beta gamma or a wrong onset fails one of the three."""
    from paper_2203_09467_b200 import workloads as W
    Ia, Ib = 823.0, 500.0
    hwp = _one_material(emo, W.PB, 1.0).material_info(0)["hwp"]                       # MeV
    onset = {I: math.sqrt(math.e) * I * 1e-6 / hwp for I in (Ia, Ib)}              # beta gamma at the onset
    for T in (0.5, 2.0, 5.0, 10.5, 11.2, 20.0, 100.0, 1e3, 1e4):
        g = T / ME + 1
        bg = math.sqrt(g * g - 1)
        b2 = 1 - 1 / (g * g)
        pa, pb = _one_material(emo, W.PB, T, I_eV=Ia), _one_material(emo, W.PB, T, I_eV=Ib)
        for kind in ("dedx_em", "dedx_ep"):
            va, vb = pa.table(0, kind)[0], pb.table(0, kind)[0]
            if bg > max(onset.values()) * (1 + 1e-9):
                assert va == pytest.approx(vb, rel=1e-12), (T, kind)
            elif bg < min(onset.values()):
                pre = 2 * math.pi * RE * RE * ME * pa.material_info(0)["n_e"] / b2
                assert vb - va == pytest.approx(pre * 2 * math.log(Ia / Ib), rel=1e-9), (T, kind)
            else:
                assert vb > va
    # the onset for I = 823 eV sits between T = 10.5 and 11.2 MeV (beta gamma = 22.2): both sides are sampled above
    assert (10.5 / ME + 1) ** 2 - 1 < onset[Ia] ** 2 < (11.2 / ME + 1) ** 2 - 1


@pytest.mark.parametrize("T,Tcut", [(10.0, 1.0), (1.0, 0.1), (1e3, 0.35), (5.0, 2.0)])
def test_restricted_loss_derivative_equals_cut_times_dcs(emo, T, Tcut):
    """d(dE/dx)_col / dT_cut = n_e T_cut dsigma/dT_delta(T_cut): ties dE/dx to the Moller/Bhabha DCS."""
    L = emo.lib()
    h = 1e-5 * Tcut
    lo = _pb_problem(emo, Tcut - h, 0.1, E_min=T, E_max=2 * T, n_E=2)
    hi = _pb_problem(emo, Tcut + h, 0.1, E_min=T, E_max=2 * T, n_E=2)
    n_e = lo.material_info(0)["n_e"]
    for kind, dcs in (("dedx_em", L.emo_moller_dcs), ("dedx_ep", L.emo_bhabha_dcs)):
        deriv = (hi.table(0, kind)[0] - lo.table(0, kind)[0]) / (2 * h)
        want = n_e * Tcut * dcs(T, Tcut / T) / T
        assert deriv == pytest.approx(want, rel=2e-6)


def test_material_constants(emo):
    from paper_2203_09467_b200 import workloads as W
    d, _ = W.config4(4)
    P = emo.Problem(d)
    # n_e [cm-3], X0 [cm], plasma energy [eV]
    want = {0: (6.99444e23, 9.3661, 31.06), 1: (2.06012e24, 0.8924, 53.30), 2: (2.34812e24, 1.4923, 56.90),
            3: (3.36476e23, 42.5411, 21.54)}
    for i, (ne, x0, hw) in want.items():
        mi = P.material_info(i)
        assert mi["n_e"] == pytest.approx(ne, rel=2e-5)
        assert mi["X0"] == pytest.approx(x0, rel=2e-4)
        assert mi["hwp"] * 1e6 == pytest.approx(hw, rel=5e-4)
    # plasma energy textbook shortcut: 28.816 eV sqrt(rho <Z/A>)
    si = P.material_info(0)
    assert si["hwp"] * 1e6 == pytest.approx(28.816 * math.sqrt(2.33 * 14 / 28.0855), rel=1e-4)


def test_gauss_legendre_nodes(emo):
    import ctypes as C
    for n in (4, 32):
        x = np.zeros(n); w = np.zeros(n)
        emo.lib().emo_gauss_legendre(n, x.ctypes.data_as(C.POINTER(C.c_double)), w.ctypes.data_as(C.POINTER(C.c_double)))
        xr, wr = np.polynomial.legendre.leggauss(n)
        assert np.allclose(x, xr, rtol=0, atol=1e-15) and np.allclose(w, wr, rtol=1e-13, atol=0)
