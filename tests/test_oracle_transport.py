"""Pins for the oracle's tables, its single step (C7) and the
transport loop (C10, C11): invariants, closed forms and brute-force re-derivations on tiny inputs."""
import ctypes as C
import math

import numpy as np
import pytest

from paper_2203_09467_b200 import workloads as W

ME = 0.51099895


@pytest.fixture(scope="module")
def pb(emo):
    desc, _ = W.config1(4)
    return desc, emo.Problem(desc)


def test_grid_lookup_is_linear_in_lnE_and_exact_at_nodes(emo, pb):
    desc, P = pb
    ph = desc["physics"]
    n = ph["n_E"]
    x = np.log(ph["E_min"]) + np.arange(n) * np.log(ph["E_max"] / ph["E_min"]) / (n - 1)
    for kind in ("compton", "pair", "dedx_em", "range_ep", "bhabha"):
        T = P.table(0, kind)
        for j in (0, 1, 17, 100, n - 2):
            assert P.lookup(0, kind, math.exp(x[j])) == pytest.approx(T[j], rel=1e-11, abs=1e-300)
            mid = math.exp(0.5 * (x[j] + x[j + 1]))
            assert P.lookup(0, kind, mid) == pytest.approx(0.5 * (T[j] + T[j + 1]), rel=1e-11, abs=1e-300)
            q = math.exp(x[j] + 0.25 * (x[j + 1] - x[j]))
            assert P.lookup(0, kind, q) == pytest.approx(0.75 * T[j] + 0.25 * T[j + 1], rel=1e-11, abs=1e-300)
        # clamped outside the grid
        assert P.lookup(0, kind, ph["E_max"] * 3) == pytest.approx(T[-1], rel=1e-12)


def test_range_tables(emo, pb):
    desc, P = pb
    ph = desc["physics"]
    n = ph["n_E"]
    E = np.exp(np.log(ph["E_min"]) + np.arange(n) * np.log(ph["E_max"] / ph["E_min"]) / (n - 1))
    for pt in ("em", "ep"):
        R, D = P.table(0, "range_" + pt), P.table(0, "dedx_" + pt)
        assert np.all(np.diff(R) > 0) and np.all(D > 0)
        assert R[0] == pytest.approx(E[0] / D[0], rel=1e-14)                 # R24
        # dR/dE = 1/dedx: trapezoid of 1/D in E agrees with the GL4 table to quadrature accuracy
        trap = np.cumsum(0.5 * (1 / D[1:] + 1 / D[:-1]) * np.diff(E))
        assert np.allclose(R[1:] - R[0], trap, rtol=2e-3)
        # forward / inverse round trip is exact to rounding
        rng = np.random.default_rng(1)
        for e in np.exp(rng.uniform(np.log(ph["E_min"]), np.log(ph["E_max"]), 200)):
            r = P.lookup(0, "range_" + pt, e)
            assert P.range_inverse(0, "range_" + pt, r) == pytest.approx(e, rel=1e-11)
        # below the grid: constant stopping power
        assert P.range_inverse(0, "range_" + pt, 0.5 * R[0]) == pytest.approx(0.5 * E[0], rel=1e-14)
    # CSDA range of a 10 MeV electron in lead is a few mm (order-of-magnitude sanity, restricted loss)
    assert 0.3 < P.lookup(0, "range_em", 10.0) < 1.5


def test_production_cuts_from_the_cut_length(emo):
    desc, _ = W.config4(4)
    P = emo.Problem(desc)
    d1, _ = W.config2(4)
    P1 = emo.Problem(d1)
    # SURVEY C5.10 (adaptive-quadrature values; grid-based values may differ in the 3rd digit)
    want = {"Pb": (1.018, 0.175), "lAr": (0.265, 0.0175), "Si": (0.406, 0.0157), "PbWO4": (0.837, 0.146),
            "brass": (0.973, 0.052), "PVT": (0.270, 0.0046)}
    got = {}
    for Pn, d in ((P, desc), (P1, d1)):
        for i, m in enumerate(d["materials"]):
            mi = Pn.material_info(i)
            got[m["name"]] = (mi["Tcut"], mi["kcut"])
    for name, (tc, kc) in want.items():
        assert got[name][0] == pytest.approx(tc, rel=5e-3), name
        assert got[name][1] == pytest.approx(kc, rel=0.08), name        # k_c snaps UP to a grid energy (spacing 6.5-7.5 %)
    # the electron cut is the energy whose unrestricted CSDA range equals the cut length
    m = dict(W.PB); m["Tcut"] = 1e9; m["kcut"] = 1e9
    dd = dict(d1); dd["materials"] = [m, W.LAR]
    Pu = emo.Problem(dd)
    assert Pu.lookup(0, "range_em", got["Pb"][0]) == pytest.approx(0.07, rel=1e-9)


def test_thresholds_in_tables(emo, pb):
    desc, P = pb
    ph = desc["physics"]; n = ph["n_E"]
    E = np.exp(np.log(ph["E_min"]) + np.arange(n) * np.log(ph["E_max"] / ph["E_min"]) / (n - 1))
    mi = P.material_info(0)
    assert np.all(P.table(0, "moller")[E <= 2 * mi["Tcut"]] == 0) and np.all(P.table(0, "moller")[E > 2.001 * mi["Tcut"]] > 0)
    assert np.all(P.table(0, "bhabha")[E <= mi["Tcut"]] == 0) and np.all(P.table(0, "bhabha")[E > 1.001 * mi["Tcut"]] > 0)
    assert np.all(P.table(0, "brems_em")[E <= mi["kcut"]] == 0) and np.all(P.table(0, "brems_em")[E > 1.001 * mi["kcut"]] > 0)
    assert np.all(P.table(0, "pair")[E <= 2 * ME] == 0)
    assert np.array_equal(P.table(0, "brems_em"), P.table(0, "brems_ep"))
    assert np.array_equal(P.table(0, "pair"), P.table(0, "pair_elem0"))


# ---------------- single step ----------------

def _track(emo, ptype, E, x=(0, 0, 50.0), u=(0, 0, 1.0), vol=0, surf=-1, prim=0, tid=0, step=0):
    t = emo.Track()
    t.x[:] = x; t.u[:] = u
    t.E = E; t.tid = tid; t.prim = prim; t.step = step; t.vol = vol; t.surf = surf; t.ptype = ptype; t.alive = 1
    return t


def _steps(emo, P, tracks, seed):
    arr = (emo.Track * len(tracks))(*tracks)
    return P.step_batch(arr, seed)


def test_photon_step_rederived_by_hand(emo, pb):
    """Photon in the Pb cube: s = -ln(xi_0)/Sigma_tot, process by xi_1, boundary wins ties (C7 steps 3-8)."""
    desc, P = pb
    L = emo.lib()
    seed = 77
    n_disc = n_bnd = 0
    for i, E in enumerate(np.geomspace(0.02, 5e3, 40)):
        tr = _track(emo, 0, E, x=(49.0, 2.0, 50.0), u=(0.6, 0.0, 0.8), prim=i, tid=1000 + i, step=3)
        r = _steps(emo, P, [tr], seed)[0]
        sig = [P.lookup(0, k, E) for k in ("compton", "photo", "pair")]
        stot = sum(sig)
        xi0 = L.emo_draw(seed, i, 1000 + i, 3, 0)
        s_int = -math.log(xi0) / stot
        d_geo = min((50 - 49.0) / 0.6, (100 - 50.0) / 0.8)
        if d_geo <= s_int:
            n_bnd += 1
            assert r.action == 3 and r.s == pytest.approx(d_geo, rel=1e-14) and r.trk.alive == 0
            assert r.escaped == E and r.n_draws == 1
        else:
            n_disc += 1
            assert r.action == 1 and r.s == pytest.approx(s_int, rel=1e-14)
            xi1 = L.emo_draw(seed, i, 1000 + i, 3, 1)
            k = 0 if xi1 * stot < sig[0] else (1 if xi1 * stot < sig[0] + sig[1] else 2)
            assert r.process == k
            assert r.trk.x[2] == pytest.approx(50 + 0.8 * s_int, rel=1e-14) if k == 0 else True
            if k == 1:      # photoelectric: photon gone, electron carries E
                assert r.trk.alive == 0 and r.n_sec == 1 and r.sec[0].ptype == 1 and r.sec[0].E == E
            if k == 0:
                assert r.trk.alive == 1 and r.trk.step == 4 and r.trk.surf == -1
                esec = r.sec[0].E if r.n_sec else r.edep
                assert r.trk.E + esec == pytest.approx(E, rel=1e-14)
            for j in range(r.n_sec):
                assert r.sec[j].tid == L.emo_child_tid(seed, i, 1000 + i, 3, r.sec_ord[j])
                assert r.sec[j].step == 0 and r.sec[j].prim == i and r.sec[j].surf == -1
                assert list(r.sec[j].x) == list(r.trk.x)
    assert n_disc > 15 and n_bnd >= 1


def test_electron_step_limits_and_loss_rederived_by_hand(emo, pb):
    desc, P = pb
    L = emo.lib()
    ph = desc["physics"]
    seed = 5
    seen = set()
    for i, E in enumerate(np.geomspace(2e-3, 5e3, 120)):
        for pt, sfx, names in ((1, "em", ("moller", "brems_em")), (2, "ep", ("bhabha", "brems_ep", "annih"))):
            tr = _track(emo, pt, E, prim=i, tid=9, step=0)
            r = _steps(emo, P, [tr], seed)[0]
            sig = [P.lookup(0, k, E) for k in names]
            stot = sum(sig)
            D, R = P.lookup(0, "dedx_" + sfx, E), P.lookup(0, "range_" + sfx, E)
            s_int = -math.log(L.emo_draw(seed, i, 9, 0, 0)) / stot if stot > 0 else math.inf
            s_loss = R if R <= ph["rho_R"] else ph["alpha_R"] * R + ph["rho_R"] * (1 - ph["alpha_R"]) * (2 - ph["rho_R"] / R)
            action = 2 if s_loss < s_int else 1
            s = min(s_int, s_loss)
            assert r.action == action and r.s == pytest.approx(s, rel=1e-14)
            if action == 2 and R <= ph["rho_R"]:
                dE = E; seen.add("stop")
            elif s * D <= ph["lin_loss"] * E:
                dE = s * D; seen.add("linear")
            else:
                dE = E - P.range_inverse(0, "range_" + sfx, R - s); seen.add("range")
            esec = sum(r.sec[j].E for j in range(r.n_sec))
            if dE == E:
                assert r.trk.alive == 0 and r.edep == pytest.approx(E, rel=1e-14)
                if pt == 2:     # positron stops: annihilation at rest, two back-to-back me photons, ordinals 2, 3
                    assert r.rest == 1 and r.n_sec == 2 and [r.sec_ord[0], r.sec_ord[1]] == [2, 3]
                    assert r.sec[0].E == ME and r.sec[1].E == ME and r.sec[0].ptype == 0
                    assert list(r.sec[0].u) == [-v for v in r.sec[1].u]
            elif action == 2:
                assert r.trk.E == pytest.approx(E - dE, rel=1e-13) and r.edep == pytest.approx(dE, rel=1e-12)
                assert r.process == -1 and r.trk.step == 1
            else:
                # energy conservation through the discrete interaction (annihilation adds 2 me)
                extra = 2 * ME if (r.process == 6 and not r.null_int) else 0.0
                if r.rest:
                    extra += 2 * ME
                assert r.trk.E + r.edep + esec == pytest.approx(E + extra, rel=1e-13)
    assert seen == {"stop", "linear", "range"}


def test_tracking_cut_kill_at_step_start(emo, pb):
    desc, P = pb
    r = _steps(emo, P, [_track(emo, 0, 5e-4), _track(emo, 2, 5e-4)], 1)
    assert r[0].trk.alive == 0 and r[0].edep == 5e-4 and r[0].below_cut == 5e-4 and r[0].n_sec == 0 and r[0].n_draws == 0
    assert r[1].trk.alive == 0 and r[1].n_sec == 2 and r[1].rest == 1 and r[1].n_draws == 2


def test_looper_cap_and_vacuum_step(emo):
    desc, _ = W.config3(4)
    P = emo.Problem(desc)
    ms = desc["physics"]["max_steps"]
    tr = _track(emo, 0, 1.0, x=(0, 0, -5.0), vol=100, step=ms - 1, u=(1.0, 0, 0))
    r = _steps(emo, P, [tr], 1)[0]
    assert r.action == 3 and r.escaped == 1.0          # photon in vacuum flies to the world boundary
    tr = _track(emo, 2, 1.0, x=(0, 0, 5.1), vol=12, step=ms - 1)
    r = _steps(emo, P, [tr], 1)[0]
    if r.trk.alive == 0 and r.looper > 0:
        assert r.looper == pytest.approx(r.trk.E + 2 * ME)


# ---------------- transport ----------------

def test_config0_energy_sum_first_collision_and_step_count(emo):
    desc, prim = W.config0()
    P = emo.Problem(desc)
    r = P.transport(prim, desc["seed"], n_threads=2, per_primary=True)
    assert r["edep"][0] == pytest.approx(1000 * 10.0, rel=1e-12)           # infinite medium: all energy deposited
    assert r["escaped"] == 0 and r["looper"] == 0
    pp = r["per_prim"]
    assert np.abs(pp[:, 0] - 10.0).max() < 1e-12
    # steps per primary = (#Compton + 1): each history ends with one photoelectric absorption or cut kill
    assert r["steps"][0] == r["inter"][0] + 1000 and r["steps"][1] == 0
    assert r["inter"][1] + 0 <= 1000 and r["tracks"].tolist() == [1000, 0, 0]
    # first-collision depth ~ Exp(Sigma_tot(10 MeV)): mean free path 7.2477 cm in Pb
    mfp = 1.0 / (P.lookup(0, "compton", 10.0) + P.lookup(0, "photo", 10.0))
    assert mfp == pytest.approx(7.2477, rel=2e-4)
    arr = (emo.Track * 1000)(*[_track(emo, 0, 10.0, x=(0, 0, 0), prim=i) for i in range(1000)])
    depth = np.array([s.s for s in P.step_batch(arr, desc["seed"])])
    assert depth.mean() == pytest.approx(mfp, rel=3 / math.sqrt(1000))
    assert np.median(depth) == pytest.approx(mfp * math.log(2), rel=0.12)


def test_step_bin_edges_by_brute_force(emo):
    """emo_step_bin against its definition written out with floats and a table: identity below 16, four equal
    sub-bins per octave above, monotone, every bin non-empty up to the overflow bin."""
    L = emo.lib()
    bins = np.array([L.emo_step_bin(n) for n in range(1, 1 << 15)])
    assert bins[:15].tolist() == list(range(1, 16))
    assert np.all(np.diff(bins) >= 0) and np.all(np.diff(bins) <= 1)
    for n in (16, 19, 20, 31, 32, 39, 40, 1000, 1023, 1024, 20000):
        e = int(math.floor(math.log2(n)))
        assert L.emo_step_bin(n) == 16 + 4 * (e - 4) + int((n - 2 ** e) / 2 ** (e - 2))
    # widths: octave e is cut into four bins of 2^(e-2) values each
    assert [int((bins == b).sum()) for b in range(16, 28)] == [4] * 4 + [8] * 4 + [16] * 4
    assert L.emo_step_bin(1 << 40) == emo.NHIST - 1 and L.emo_step_bin(0) == 0


def test_steps_per_track_histogram_config0(emo):
    """Config 0 has one track per primary (photons only, electrons deposited at creation), so the histogram
    of steps per track must be the histogram of the per-primary step counts, which come from another counter."""
    desc, prim = W.config0()
    P = emo.Problem(desc)
    r = P.transport(prim, desc["seed"], n_threads=2, per_primary=True)
    per_primary = r["per_prim"][:, 5].astype(np.int64)
    assert per_primary.max() < 16                                          # identity bins: n itself
    want = np.bincount(per_primary, minlength=emo.NHIST)
    assert np.array_equal(r["step_hist"][0], want.astype(np.uint64))
    assert r["step_hist"][1:].sum() == 0
    assert int((np.arange(emo.NHIST) * r["step_hist"][0]).sum()) == int(r["steps"][0])


@pytest.mark.parametrize("cfg,n", [(1, 40), (2, 6), (3, 6), (4, 24), (5, 60), (6, 24)])
def test_energy_closure_per_event(emo, cfg, n):
    desc, prim = W.get(cfg, n)
    P = emo.Problem(desc)
    r = P.transport(prim, desc["seed"], per_primary=True)
    pp = r["per_prim"]
    closure = np.abs(pp[:, 0] + pp[:, 1] + pp[:, 2] - pp[:, 4]) / pp[:, 4]
    assert closure.max() < 1e-9                                            # B:north_star
    assert r["edep"].sum() + r["escaped"] + r["looper"] == pytest.approx(r["E_in"], rel=1e-11)
    assert np.allclose(r["per_prim_tally"].sum(0), r["edep"], rtol=1e-12)
    assert r["track_steps"] == int(r["steps"].sum()) == int(pp[:, 5:8].sum())
    assert r["tracks"].tolist() == pp[:, 8:11].sum(0).astype(int).tolist()
    # steps-per-track histogram: one entry per track; the mean steps per track lies inside the bins' bounds
    assert r["step_hist"].sum(1).tolist() == r["tracks"].tolist()
    lo = np.array([b if b < 16 else (4 + (b - 16) % 4) << ((b - 16) // 4 + 2) for b in range(emo.NHIST)], dtype=np.float64)
    hi = np.array([lo[b + 1] - 1 if b + 1 < emo.NHIST else np.inf for b in range(emo.NHIST)])
    for k in range(3):
        assert (lo * r["step_hist"][k]).sum() <= r["steps"][k] <= (np.where(r["step_hist"][k] > 0, hi, 0) * r["step_hist"][k]).sum()
    # every e+ ends by annihilation (in flight or at rest) unless it escaped or looped
    if r["escaped"] == 0 and r["looper"] == 0:
        assert r["tracks"][2] == r["inter"][6] + r["inter"][7]
    if cfg == 1:
        assert r["escaped"] / r["E_in"] < 0.01                            # 1 m of Pb contains a 1 GeV shower


def test_histories_do_not_depend_on_threading_or_batching(emo):
    desc, prim = W.config2(8)
    P = emo.Problem(desc)
    a = P.transport(prim, 2, n_threads=1, per_primary=True)
    b = P.transport(prim, 2, n_threads=4, per_primary=True)
    assert np.array_equal(a["per_prim"], b["per_prim"]) and np.array_equal(a["per_prim_tally"], b["per_prim_tally"])
    # a prefix of the primaries reproduces the same histories (keyed RNG, C2)
    c = P.transport(W.prefix(prim, 3), 2, n_threads=2, per_primary=True)
    assert np.array_equal(a["per_prim"][:3], c["per_prim"])
    # a different seed gives different histories
    d = P.transport(W.prefix(prim, 3), 3, n_threads=2, per_primary=True)
    assert not np.array_equal(c["per_prim"], d["per_prim"])


def test_shower_sanity_config2(emo):
    """Order-of-magnitude physics sanity (parity unpinned beyond conservation)."""
    desc, prim = W.config2(12)
    P = emo.Problem(desc)
    r = P.transport(prim, 2, per_primary=True)
    prof = r["edep"].reshape(50, 2).sum(1)
    zmax = (np.argmax(prof) + 0.5) * 0.8
    # shower maximum near ln(E/Ec) X0_eff: a 10 GeV shower in this stack peaks a few cm deep
    assert 2.0 < zmax < 12.0
    frac_ar = r["edep"][1::2].sum() / r["edep"].sum()
    assert 0.05 < frac_ar < 0.5                                            # sampling fraction of lAr


def test_paper_verification_problem_geometry(emo):
    """SURVEY 8(f) f1 / PAPER.md:172-176: six cylindrical regions to 375 cm cut into z slabs.  A straight
    radial photon crosses the shells at the declared radii, and the slab tallies of a small run add up to
    the deposited energy (the z tally lives in the geometry)."""
    desc, prim = W.get(5, 40)
    P = emo.Problem(desc)
    x, u, vol, surf = np.array([0.0, 0.0, 3.0]), np.array([1.0, 0.0, 0.0]), 0, -1
    radii = []
    for _ in range(6):
        d, hit = P.distance(vol, x, u, surf)
        x = x + d * u
        radii.append(float(np.hypot(x[0], x[1])))
        vol, surf = P.neighbour(x, u, hit), hit
        if vol < 0:
            break
    assert radii == pytest.approx([30.0, 125.0, 175.0, 275.0, 325.0, 375.0], abs=1e-9) and vol == -1
    r = P.transport(prim, desc["seed"], per_primary=True)
    assert len(r["edep"]) == 28
    assert r["edep"].sum() + r["escaped"] + r["looper"] == pytest.approx(r["E_in"], rel=1e-11)
    assert r["edep"][13] + r["edep"][14] > 0.4 * r["E_in"]            # isotropic source: most energy near z = 0


def test_longitudinal_shower_profile_of_1_gev_electrons_in_lead(emo):
    """Shower shape pinned by what cascade theory and the PDG review fix (SURVEY C13 keeps the
    rest of the aggregate physics "parity unpinned"): in units of the radiation length t = z / X0 the longitudinal
    profile of an electron-induced shower peaks at t_max = ln(E / E_c) - 0.5 with E_c = 610 MeV / (Z + 1.24)
    (PDG, "Passage of particles through matter", electromagnetic cascades: Rossi's critical energy for solids and the
    shower-maximum rule), and 95 % of the energy lies within t_max + 0.08 Z + 9.6 radiation lengths (same review,
    longitudinal containment).  300 showers of 1 GeV in 60 lead slabs of X0 / 2, 1 m wide."""
    X0 = emo.Problem(W.config1(1)[0]).material_info(0)["X0"]
    nz, dz = 60, 0.5 * X0
    surfaces = [(W.PX, -50.0), (W.PX, 50.0), (W.PY, -50.0), (W.PY, 50.0)] + [(W.PZ, k * dz) for k in range(nz + 1)]
    volumes = [dict(surf=[0, 1, 2, 3, 4 + k, 5 + k], sense=[1, -1, 1, -1, 1, -1], material=0, tally=k) for k in range(nz)]
    desc = dict(name="pb_slabs", seed=11, materials=[W.PB], surfaces=surfaces, volumes=volumes, field=(0.0, 0.0, 0.0),
                physics=W.physics(), n_slots=1 << 16, queue_capacity=1 << 20)
    n = 300
    prim = W._prim(n, 1, 1000.0, (0, 0, 0), (0, 0, 1), 0, 4)
    r = emo.Problem(desc).transport(prim, 11)
    prof = r["edep"] / r["edep"].sum()
    assert r["edep"].sum() + r["escaped"] == pytest.approx(r["E_in"], rel=1e-9)
    assert r["escaped"] / r["E_in"] < 0.01                                # 30 X0 deep, 1 m wide
    t = (np.arange(nz) + 0.5) * 0.5                                       # slab centres in radiation lengths
    Ec = 610.0 / (82 + 1.24)
    t_max = math.log(1000.0 / Ec) - 0.5                                   # 4.41
    # maximum of the profile: vertex of the parabola through the highest slab and its neighbours
    k = int(np.argmax(prof))
    y0, y1, y2 = prof[k - 1], prof[k], prof[k + 1]
    peak = t[k] + 0.5 * 0.5 * (y0 - y2) / (y0 - 2 * y1 + y2)
    assert abs(peak - t_max) < 1.0, (peak, t_max)
    # a gamma-distribution profile t^(a-1) e^(-b t) with b = 0.5 (lead, 1 GeV) has its mean 1 / b beyond the maximum
    mean = float((t * prof).sum())
    assert t_max + 1.0 < mean < t_max + 3.5, (mean, t_max)
    L95 = t_max + 0.08 * 82 + 9.6                                         # 20.6 X0
    inside = float(prof[t < L95].sum())
    assert 0.92 < inside < 0.99, inside
    # and the profile rises to its maximum and falls after it (smoothed over 3 slabs: 300 showers fluctuate)
    sm = np.convolve(prof, np.ones(3) / 3, mode="valid")
    ks = int(np.argmax(sm))
    assert np.all(np.diff(sm[:ks + 1]) > 0) and np.all(np.diff(sm[ks + 3:ks + 30]) < 0)
