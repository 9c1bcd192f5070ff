"""-m gpu: the CUDA path, called through the C-ABI (paper_2203_09467_b200.emx -> libemx.so), against the
oracle on the same seeded inputs.  Levels follow BASELINE.json north_star: (1) integer / indexing work
bit-exact, (2) single-step outputs on identical fp64 states to 1e-12, (3) aggregate observables within
3 standard errors and 1e-3 relative; plus energy closure to 1e-9.
"""
import numpy as np
import pytest

from conftest import golden
from paper_2203_09467_b200 import workloads as W
import states

pytestmark = pytest.mark.gpu

RTOL2 = states.RTOL2   # level 2 (north_star)


@pytest.fixture(scope="module")
def emx():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2203_09467_b200 import emx as m
    m.lib()
    return m


# ---------------- level 1: integer work ----------------

def test_philox_known_answers_and_draws(emx, emo):
    rows = golden("philox4x32_10_kat.txt")
    ctr = np.array([[int(x, 16) for x in r[0:4]] for r in rows], dtype=np.uint32)
    key = np.array([[int(x, 16) for x in r[4:6]] for r in rows], dtype=np.uint32)
    want = np.array([[int(x, 16) for x in r[6:10]] for r in rows], dtype=np.uint32)
    assert np.array_equal(emx.philox_batch(ctr, key), want)
    rng = np.random.default_rng(0)
    n = 5000
    prim = rng.integers(0, 2 ** 32, n, dtype=np.uint64).astype(np.uint32)
    tid = rng.integers(0, 2 ** 63, n, dtype=np.uint64)
    step = rng.integers(0, 10000, n, dtype=np.uint64).astype(np.uint32)
    nn = rng.integers(0, 40, n, dtype=np.uint64).astype(np.uint32)
    u, ch = emx.draw_batch(12345, prim, tid, step, nn)
    L = emo.lib()
    u_ref = np.array([L.emo_draw(12345, int(prim[i]), int(tid[i]), int(step[i]), int(nn[i])) for i in range(n)])
    c_ref = np.array([L.emo_child_tid(12345, int(prim[i]), int(tid[i]), int(step[i]), int(nn[i])) for i in range(n)],
                     dtype=np.uint64)
    assert np.array_equal(u, u_ref) and np.array_equal(ch, c_ref)      # bit-exact
    assert u.min() > 0.0 and u.max() < 1.0


def _refill_reference(alive, capacity, n_queue):
    """Trivial CPU statement of the refill rule: hole k (ascending) <- record
    [q-1-k]; stack dry -> j-th live track from the end moves into the j-th remaining hole below the new
    range; surplus records are appended above the old range."""
    n_old = len(alive)
    src = np.full(capacity, -1, dtype=np.int32)
    holes = [i for i in range(n_old) if not alive[i]]
    h, q = len(holes), n_queue
    a = min(h, q)
    for k in range(a):
        src[holes[k]] = q - 1 - k
    n_new = n_old - (h - a)
    rest = [i for i in holes[a:] if i < n_new]
    movers = [i for i in range(n_old - 1, n_new - 1, -1) if alive[i]]
    assert len(rest) == len(movers)
    for j, i in enumerate(movers):
        src[rest[j]] = -2 - i
    extra = min(q - a, capacity - n_old) if h == a else 0
    for k in range(extra):
        src[n_old + k] = q - 1 - a - k
    return src, (n_new + extra, q - a - extra, h - a)


@pytest.mark.parametrize("n_live,capacity,n_queue,p_dead", [
    (0, 1000, 0, 0.0), (0, 1000, 300, 0.0), (0, 300, 1000, 0.0), (777, 1024, 0, 0.3), (777, 1024, 50, 0.3),
    (777, 1024, 5000, 0.3), (1024, 1024, 100, 1.0), (5000, 8192, 700, 0.5), (5000, 8192, 10 ** 6, 0.02),
    (100003, 131072, 999, 0.7), (100003, 131072, 0, 0.999), (129, 256, 3, 0.9)])
def test_refill_compaction_order_is_bit_exact(emx, n_live, capacity, n_queue, p_dead):
    rng = np.random.default_rng(n_live + n_queue)
    alive = (rng.random(n_live) >= p_dead).astype(np.uint8)
    src, counts = emx.refill_plan(alive, capacity, n_queue)
    ref, rc = _refill_reference(alive, capacity, n_queue)
    assert counts == rc
    assert np.array_equal(src[:rc[0]], ref[:rc[0]])
    # every slot of the new live range is live: untouched live track, queue record or moved track
    n_new = rc[0]
    live_after = np.array([(i < n_live and alive[i]) or src[i] != -1 for i in range(n_new)], dtype=bool)
    assert live_after.all()
    used = src[:n_new][src[:n_new] >= 0]
    assert len(np.unique(used)) == len(used)                          # no record handed out twice


# ---------------- tables ----------------

def _workload(cfg, n):
    """W.get (config 7 = calorimeter with multiple scattering and energy-loss fluctuations), plus 37 = config 3
    (calorimeter in a 1 T field) with multiple scattering alone, 47 = config 4 (barrel, 4 T) with both -- the deflection
    at the end of a curved step -- and 17 = config 1 (Pb cube) with the fluctuations alone; 27 / 38 / 48 = configs 2 / 3 / 4
    with the spatial moments of multiple scattering as well (msc = 2, DESIGN.md R-MSC2: path-length correction and
    lateral displacement), with / without / with fluctuations"""
    ext = {37: dict(msc=1, msc_fr=0.2, msc_smin=1e-3), 47: dict(msc=1, msc_fr=0.1, msc_smin=2e-3, fluct=1), 17: dict(fluct=1),
           27: dict(msc=2, msc_fr=0.2, msc_smin=1e-3, fluct=1), 38: dict(msc=2, msc_fr=0.2, msc_smin=1e-3),
           48: dict(msc=2, msc_fr=0.1, msc_smin=2e-3, fluct=1),
           43: dict(integrator=1), 63: dict(integrator=1),      # the Dormand-Prince integrator (R-INT): barrel at 4 T, fringe field
           49: dict(msc=2, msc_fr=0.1, msc_smin=2e-3, fluct=1, integrator=1)}   # everything optional at once
    if cfg in ext:
        desc, prim = W.get(cfg // 10, n)
        desc = dict(desc, physics=dict(desc["physics"], **ext[cfg]), seed=cfg)
        return desc, prim
    return W.get(cfg, n)


@pytest.mark.parametrize("cfg", [0, 1, 2, 4, 7, 17, 47, 27, 48])
def test_tables_match_the_oracle(emx, emo, cfg):
    desc, _ = _workload(cfg, 4)
    G, O = emx.Problem(desc), emo.Problem(desc)
    worst = 0.0
    for im in range(len(desc["materials"])):
        for kind in emx.T_NAMES:
            a, b = O.table(im, kind), G.table(im, kind)
            assert np.array_equal(a == 0, b == 0), (im, kind)      # thresholds fall on the same grid points
            nz = a != 0
            if nz.any():
                worst = max(worst, float(np.max(np.abs(a[nz] - b[nz]) / np.abs(a[nz]))))
        mo, mg = O.material_info(im), G.material_info(im)
        for k in ("n_e", "I", "hwp", "X0", "Tcut", "kcut"):
            assert mg[k] == pytest.approx(mo[k], rel=1e-13), (im, k)
    assert worst <= RTOL2, worst


# ---------------- level 2: single step ----------------

@pytest.mark.parametrize("cfg,n", [(0, 20000), (1, 40000), (2, 40000), (3, 40000), (4, 40000), (5, 20000), (6, 40000),
                                   (7, 40000), (17, 40000), (37, 40000), (47, 40000), (27, 40000), (38, 40000), (48, 40000), (43, 40000), (63, 40000), (49, 40000)])
def test_single_step_parity(emx, emo, cfg, n):
    desc, _ = _workload(cfg, 4)
    G, O = emx.Problem(desc), emo.Problem(desc)
    tr = states.random_states(emo, O, desc, n, seed=1000 + cfg)
    ref = states.result_arrays(O.step_batch(tr, desc["seed"]))
    gin = (emx.Track * n).from_buffer_copy(bytes(tr))
    got = states.result_arrays(G.step_batch(gin, desc["seed"]))
    E_in = np.array([t.E for t in tr])
    # level 1: action, process, secondary counts and ids, draw counts, cells, substep counts: bit-exact on every state
    # level 2: 1e-12 (north_star) for every step without field substeps; a field step is held to the bound derived
    # from its own substep count, a step with fluctuated loss to 1e-12 E / E' (states.step_tolerances)
    tol = states.step_tolerances(desc, tr, ref)
    n_bad, worst, rep = states.compare_steps(ref, got, E_in, tol)
    assert n_bad == 0, rep
    assert worst <= 1.0, {k: v for k, v in rep.items() if isinstance(v, float) and v > 0.5}
    plain = (ref["n_sub"] == 0) & (tol["E"] == states.RTOL2)      # the plain 1e-12 of north_star holds for these
    assert plain.sum() > n // 4 and np.all(tol["u"][plain] == states.RTOL2) and np.all(tol["x"][plain] == states.RTOL2)
    if cfg in (3, 4, 6, 37, 47, 38, 48, 43, 63, 49):
        assert tol["trunc"].sum() <= n // 6 and (ref["n_sub"] > 1).sum() > n // 10
    # coverage of the branches
    acts = np.bincount(ref["action"], minlength=6)
    assert acts[1] > 0 and (cfg == 0 or acts[3] > 0)
    fl = desc["physics"]["fluct"]
    if cfg in (7, 37, 47, 27, 38, 48, 49):      # multiple scattering: the step limit was hit, deflections happened before interactions
        assert acts[5] > 0 and (ref["msc_tau"][ref["action"] == 1] > 0).any() and (ref["msc_tau"][ref["action"] == 3] > 0).any()
        assert np.all(ref["n_draws"][(ref["msc_tau"] > 0) & (ref["action"] == 1)] >= 4 + 2 * fl)
    else:
        assert acts[5] == 0 and not ref["msc_tau"].any()
    if fl:                      # fluctuations: charged steps in matter without an interaction drew three numbers (+ 2 for msc)
        pt = np.array([t.ptype for t in tr])
        m = (pt != 0) & np.isin(ref["action"], (2, 3, 5)) & (ref["alive"] == 1) & (ref["edep"] > 0)
        assert m.sum() > 100 and np.all(ref["n_draws"][m] == 3 + 2 * (desc["physics"]["msc"] > 0))


# ---------------- level 3: transport ----------------

def _per_primary_se(o):
    """standard errors of the per-primary means from the oracle run"""
    n = o["per_prim"].shape[0]
    return o["per_prim_tally"].std(axis=0, ddof=1) / np.sqrt(n), o["per_prim"].std(axis=0, ddof=1) / np.sqrt(n)


@pytest.mark.parametrize("integrator", [0, 1])
@pytest.mark.parametrize("field,fringe", [((0.0, 1.0, 0.0), None), ((0.0, 0.0, -4.0), None), ((1.0, -2.0, 0.5), None),
                                          ((0.0, 0.0, 3.8), (120.0, 15.0))])
def test_one_field_substep_at_1e_12(emx, emo, field, fringe, integrator):
    """Level 2 for ONE substep of the propagation: rk4_doubling (integrator 0) and the Dormand-Prince
    step (integrator 1) of the kernel (axis-specialised for a field along +-x, +-y, +-z; general; field map) against the
    oracle's, state by state.  One substep is a
    fixed sequence of IEEE operations on both sides, so 1e-12 holds without any allowance: positions relative to
    max(|x|, h), directions absolute (unit vectors), and the error estimate -- a DIFFERENCE of two positions, so its
    rounding is that of the positions -- absolute on the same scale."""
    desc, _ = W.get(4, 4)
    desc = dict(desc, field=field, physics=dict(desc["physics"], integrator=integrator))
    if fringe:
        desc["field_fringe"] = fringe
    G, O = emx.Problem(desc), emo.Problem(desc)
    rng = np.random.default_rng(99)
    n = 20000
    x = rng.uniform(-150.0, 150.0, size=(n, 3))
    u = rng.normal(size=(n, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    pmom = 10.0 ** rng.uniform(-1.5, 5.0, size=n)                     # MeV/c
    kappa = np.where(rng.random(n) < 0.5, -1.0, 1.0) * 2.99792458 * float(np.linalg.norm(field)) / pmom
    h = np.minimum(0.25 / np.abs(kappa), 10.0 ** rng.uniform(-6.0, 2.0, size=n)) * rng.choice([1.0, 0.37, 0.05], size=n)
    x1, u1, err = emx.field_substep_batch(G, x, u, kappa, h)
    L = emo.lib()
    import ctypes as C
    dp = C.POINTER(C.c_double)
    ox, ou, oe = np.empty((n, 3)), np.empty((n, 3)), np.empty(n)
    Bhat = np.array(field) / np.linalg.norm(field)
    e = C.c_double()
    for i in range(n):
        a = (x[i].ctypes.data_as(dp), u[i].ctypes.data_as(dp))
        o = (ox[i].ctypes.data_as(dp), ou[i].ctypes.data_as(dp), C.byref(e))
        if integrator == 1:
            L.emo_dp45(O.h, a[0], a[1], kappa[i], h[i], *o)
        elif fringe:
            L.emo_rk4_doubling_map(O.h, a[0], a[1], kappa[i], h[i], *o)
        else:
            L.emo_rk4_doubling(a[0], a[1], kappa[i], Bhat.ctypes.data_as(dp), h[i], *o)
        oe[i] = e.value
    scale = np.maximum(np.linalg.norm(x, axis=1), h)
    assert np.max(np.linalg.norm(x1 - ox, axis=1) / scale) <= 1e-12
    assert np.max(np.abs(u1 - ou)) <= 1e-12
    assert np.max(np.abs(err - oe) / scale) <= 1e-12
    assert np.all(np.abs(np.linalg.norm(u1, axis=1) - 1.0) < 4e-16)
    assert (oe > 1e-7).sum() > n // 50 and (oe < 1e-7).sum() > n // 4     # rejected and accepted substeps both occur


@pytest.mark.parametrize("cfg,n,n_slots", [(0, 1000, 1024), (1, 300, 1 << 16), (2, 24, 1 << 16), (3, 24, 1 << 16),
                                           (4, 48, 1 << 16), (1, 64, 1024), (5, 400, 1 << 16), (6, 48, 1 << 16),
                                           (7, 24, 1 << 16), (17, 300, 1 << 16), (37, 24, 1 << 16), (47, 48, 1 << 16),
                                           (27, 24, 1 << 16), (48, 48, 1 << 16), (43, 48, 1 << 16), (49, 48, 1 << 16)])
def test_transport_parity_and_energy_closure(emx, emo, cfg, n, n_slots):
    desc, prim = _workload(cfg, n)
    G, O = emx.Problem(desc), emo.Problem(desc)
    o = O.transport(prim, desc["seed"], per_primary=True)
    g = G.transport(G.upload_primaries(prim), desc["seed"], n_slots=n_slots, queue_capacity=1 << 20)
    # energy closure (north_star: 1e-9 relative)
    assert g["E_in"] == pytest.approx(o["E_in"], rel=1e-14)
    assert g["edep"].sum() + g["escaped"] + g["looper"] == pytest.approx(g["E_in"], rel=1e-9)
    # level 3: means per primary within 3 standard errors AND 1e-3 relative (common random numbers)
    se_t, se_p = _per_primary_se(o)
    mean_o, mean_g = o["edep"] / n, g["edep"] / n
    big = mean_o > 1e-6 * o["E_in"] / n
    assert np.all(np.abs(mean_g - mean_o) <= 3 * se_t + 1e-12 * np.abs(mean_o) + 1e-300)   # + summation rounding
    assert np.all(np.abs(mean_g[big] - mean_o[big]) <= 1e-3 * mean_o[big])
    for k in ("escaped", "below_cut", "looper"):
        assert abs(g[k] - o[k]) <= 1e-3 * max(abs(o[k]), 1e-6 * o["E_in"]), k
    for k in ("steps", "tracks", "inter"):
        a, b = o[k].astype(np.float64), g[k].astype(np.float64)
        assert np.all(np.abs(a - b) <= 1e-3 * np.maximum(a, 1.0) + 3.0), (k, o[k], g[k])
    assert g["track_steps"] == int(g["steps"].sum())
    assert g["stalls"] == 0
    # steps-per-track histogram: one entry per track; bins within 3 sigma (Poisson) and 1e-3
    hg, ho = G.read_step_hist(), o["step_hist"]
    assert hg.sum(1).tolist() == g["tracks"].tolist()
    a, b = ho.astype(np.float64), hg.astype(np.float64)
    assert np.all(np.abs(a - b) <= 1e-3 * a + 3.0 * np.sqrt(np.maximum(a, 1.0)) * (a != b)), (ho, hg)
    if cfg == 0:
        assert g["edep"][0] == pytest.approx(1000 * 10.0, rel=1e-12)
        assert np.array_equal(g["steps"], o["steps"]) and np.array_equal(g["inter"], o["inter"])
    if np.array_equal(g["steps"], o["steps"]) and np.array_equal(g["tracks"], o["tracks"]):
        assert np.array_equal(hg, ho)                  # same histories step for step: the same histogram


def test_full_stack_stalls_do_not_change_the_physics(emx, emo):
    """R7: with a tiny stack the loop throttles instead of overflowing, and the result is the same."""
    desc, prim = W.get(1, 48)
    G = emx.Problem(desc)
    pd = G.upload_primaries(prim)
    a = G.transport(pd, desc["seed"], n_slots=4096, queue_capacity=1 << 20)
    b = G.transport(pd, desc["seed"], n_slots=4096, queue_capacity=3000)
    assert b["stalls"] > 0 and a["stalls"] == 0
    assert np.array_equal(a["steps"], b["steps"]) and np.array_equal(a["inter"], b["inter"])
    assert np.array_equal(a["tracks"], b["tracks"])
    assert b["edep"].sum() == pytest.approx(a["edep"].sum(), rel=1e-12)
    assert b["peak_queue"] <= 3000 * 1.01 + 384
    hb = G.read_step_hist()
    G.transport(pd, desc["seed"], n_slots=4096, queue_capacity=1 << 20)
    assert np.array_equal(hb, G.read_step_hist())      # stalled steps are not counted twice


@pytest.mark.parametrize("case", ["none", "one", "escape_at_once", "positrons_below_cut", "photons_below_cut", "grid_top"])
def test_degenerate_primaries_against_the_oracle(emx, emo, case):
    """Edge cases of the loop: no primary, one primary, primaries that leave the world in their first step,
    primaries born below the tracking cut (e+ still annihilate at rest), energies at the top of the grid."""
    desc, prim = W.get(4, 16)
    p = {k: v.copy() for k, v in prim.items()}
    if case == "none":
        p = {k: v[:0] for k, v in p.items()}
    elif case == "one":
        p = {k: v[:1] for k, v in p.items()}
    elif case == "escape_at_once":
        p["pos"][:, 2] = 149.99
        p["dir"][:] = np.array([0.0, 0.0, 1.0])
    elif case == "positrons_below_cut":
        p["ptype"][:] = 2
        p["E"][:] = 0.0005
    elif case == "photons_below_cut":
        p["ptype"][:] = 0
        p["E"][:] = 0.0005
    elif case == "grid_top":
        p = {k: v[:2] for k, v in p.items()}
        p["E"][:] = 1e5
    G, O = emx.Problem(desc), emo.Problem(desc)
    o = O.transport(p, desc["seed"])
    g = G.transport(G.upload_primaries(p), desc["seed"], n_slots=1 << 14, queue_capacity=1 << 21)
    assert g["E_in"] == pytest.approx(o["E_in"], rel=1e-14, abs=0.0)
    for k in ("steps", "tracks", "inter"):
        a, b = o[k].astype(np.float64), g[k].astype(np.float64)
        assert np.all(np.abs(a - b) <= 1e-3 * a + 3.0), (k, o[k], g[k])
    if case in ("none", "escape_at_once", "positrons_below_cut", "photons_below_cut"):
        assert np.array_equal(g["steps"], o["steps"]) and np.array_equal(g["tracks"], o["tracks"])
        assert np.array_equal(G.read_step_hist(), o["step_hist"])
    for k in ("escaped", "below_cut", "looper"):
        assert g[k] == pytest.approx(o[k], rel=1e-3, abs=1e-9), k
    assert g["edep"].sum() == pytest.approx(o["edep"].sum(), rel=1e-3, abs=1e-9)
    assert g["stalls"] == 0


def test_hopelessly_small_workspace_is_an_error_not_a_hang(emx):
    """R7: 100 GeV showers in 384 slots with 1000 stack records dead-lock (every live track waits for room on a
    full stack, and stalled warps keep pushing and retiring tombstones).  The loop must notice that no step is
    committed any more and return EMX_E_CAPACITY; the same problem with room runs."""
    desc, prim = W.get(4, 8)
    G = emx.Problem(desc)
    pd = G.upload_primaries(prim)
    with pytest.raises(emx.EmxError, match="-4"):
        G.transport(pd, desc["seed"], n_slots=384, queue_capacity=1000)
    ok = G.transport(pd, desc["seed"], n_slots=384, queue_capacity=1 << 20)
    assert ok["stalls"] == 0 and ok["track_steps"] > 100000
    assert ok["edep"].sum() + ok["escaped"] + ok["looper"] == pytest.approx(ok["E_in"], rel=1e-9)


def test_arena_smaller_than_a_wave_of_primaries_ends(emx):
    """a wave of primaries used to be admitted whole or not at all, so an arena smaller than the wave spun
    in the graph's WHILE node for ever.  Waves are clipped to the room of the arena now: the run ends -- with the same
    histories as a roomy run when the slots can absorb the showers (stalled interactions are retried, R7), or with
    EMX_E_CAPACITY when nothing moves any more."""
    desc, prim = W.get(1, 600)                                        # 600 primaries, 200 records
    G = emx.Problem(desc)
    pd = G.upload_primaries(prim)
    roomy = G.transport(pd, desc["seed"], n_slots=1 << 16, queue_capacity=1 << 20)
    try:
        r = G.transport(pd, desc["seed"], n_slots=1 << 16, queue_capacity=200)
    except emx.EmxError as e:
        assert "-4" in str(e)
    else:
        assert r["peak_queue"] <= 200 + 384
        for k in ("steps", "tracks", "inter"):
            assert np.array_equal(r[k], roomy[k]), k
        assert r["edep"].sum() + r["escaped"] + r["looper"] == pytest.approx(r["E_in"], rel=1e-9)
    desc0, prim0 = W.get(0, 1000)                                     # photons that queue no secondaries: 1000 through 64 records
    G0 = emx.Problem(desc0)
    r = G0.transport(G0.upload_primaries(prim0), desc0["seed"], n_slots=1024, queue_capacity=64)
    assert r["tracks"][0] == 1000 and r["peak_queue"] <= 64
    assert r["edep"].sum() + r["escaped"] == pytest.approx(r["E_in"], rel=1e-9)


def test_rebuilding_after_a_changed_production_cut_equals_a_fresh_problem(emx):
    """the production thresholds derived from prod_cut_cm belong to the build, not to the problem: build,
    change the cut length, rebuild -> thresholds and every table equal those of a problem created with the new cut."""
    import ctypes as C
    desc, _ = W.get(2, 4)
    G = emx.Problem(desc)
    old = [G.material_info(m)["Tcut"] for m in range(2)]
    ph = emx.Physics()
    for k, _ in emx.Physics._fields_:
        setattr(ph, k, desc["physics"][k])
    ph.prod_cut_cm = 0.2
    G._check(emx.lib().emx_set_physics(G.h, C.byref(ph)))
    G.build_tables()
    fresh = emx.Problem(dict(desc, physics=dict(desc["physics"], prod_cut_cm=0.2)))
    for m in range(2):
        a, b = G.material_info(m), fresh.material_info(m)
        assert a["Tcut"] == b["Tcut"] and a["kcut"] == b["kcut"]
        assert a["Tcut"] > 1.5 * old[m]                               # the cut did change
        for kind in emx.T:
            assert np.array_equal(G.table(m, kind), fresh.table(m, kind)), (m, kind)


def test_transport_on_a_side_stream_is_ordered_after_the_work_queued_on_it(emx):
    """The `stream` argument: primaries uploaded on a non-default torch stream are consumed by a transport on
    that same stream without any synchronisation in between (the library's internal streams are ordered after
    the caller's stream, and the caller's stream after them)."""
    import torch
    desc, prim = W.get(2, 12)
    G = emx.Problem(desc)
    ref = G.transport(G.upload_primaries(prim), desc["seed"], n_slots=1 << 13, queue_capacity=1 << 18)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        pd = G.upload_primaries(prim)
        a = G.transport(pd, desc["seed"], n_slots=1 << 13, queue_capacity=1 << 18)
        b = G.transport_host(prim, desc["seed"], n_slots=1 << 13, queue_capacity=1 << 18)
    for r in (a, b):
        assert np.array_equal(r["steps"], ref["steps"]) and np.array_equal(r["inter"], ref["inter"])
        assert np.allclose(r["edep"], ref["edep"], rtol=1e-11, atol=1e-9)


def test_results_do_not_depend_on_slots_or_host_entry(emx):
    desc, prim = W.get(2, 12)
    G = emx.Problem(desc)
    a = G.transport(G.upload_primaries(prim), desc["seed"], n_slots=1 << 12, queue_capacity=1 << 18)
    b = G.transport_host(prim, desc["seed"], n_slots=1 << 15, queue_capacity=1 << 18)
    assert np.array_equal(a["steps"], b["steps"]) and np.array_equal(a["tracks"], b["tracks"])
    assert np.allclose(a["edep"], b["edep"], rtol=1e-11, atol=1e-9)
    assert a["iterations"] != b["iterations"] or a["peak_live"] != b["peak_live"]
    # nor on how many slots there are for the two pools to share (256: one chunk each; the pools trade chunks)
    c = G.transport(G.upload_primaries(prim), desc["seed"], n_slots=256, queue_capacity=1 << 18)
    assert np.array_equal(a["steps"], c["steps"]) and np.array_equal(a["tracks"], c["tracks"])
    assert np.array_equal(a["inter"], c["inter"])
    assert np.allclose(a["edep"], c["edep"], rtol=1e-11, atol=1e-9)
    assert c["peak_live"] <= 256 and c["iterations"] > a["iterations"]


def test_shards_of_the_primaries_sum_to_the_whole(emx):
    """the primaries cut into contiguous parts, each transported with its offset (here one after
    the other on one GPU, as the ranks of a sharded job would), give the counters of the whole list exactly and
    its tallies up to summation order."""
    from paper_2203_09467_b200 import shard
    desc, prim = W.get(3, 16)
    G = emx.Problem(desc)
    whole = G.transport(G.upload_primaries(prim), desc["seed"], n_slots=1 << 14, queue_capacity=1 << 20)
    h_whole = G.read_step_hist()
    parts, hists = [], []
    for rank in range(3):
        first, sub = shard.shard_primaries(prim, rank, 3)
        G.set_primary_offset(first)
        parts.append(G.transport(G.upload_primaries(sub), desc["seed"], n_slots=1 << 14, queue_capacity=1 << 20))
        hists.append(G.read_step_hist())
    G.set_primary_offset(0)
    for k in ("steps", "tracks", "inter"):
        assert np.array_equal(sum(p[k].astype(np.int64) for p in parts), whole[k].astype(np.int64)), k
    assert sum(p["null_int"] for p in parts) == whole["null_int"]
    assert np.array_equal(sum(h.astype(np.int64) for h in hists), h_whole.astype(np.int64))
    assert np.allclose(sum(p["edep"] for p in parts), whole["edep"], rtol=1e-11, atol=1e-9)
    assert sum(p["E_in"] for p in parts) == pytest.approx(whole["E_in"], rel=1e-14)
    # without the offsets the parts are different histories
    first, sub = shard.shard_primaries(prim, 2, 3)
    other = G.transport(G.upload_primaries(sub), desc["seed"], n_slots=1 << 14, queue_capacity=1 << 20)
    assert not np.array_equal(other["steps"], parts[2]["steps"])
    with pytest.raises(emx.EmxError):
        G.set_primary_offset(-1)


def test_kept_iteration_graph_is_dropped_when_an_argument_changes(emx):
    """emx_transport keeps the instantiated graph for the next call with the same kernel arguments; a new seed,
    new primaries, another workspace size or rebuilt tables must each give the result of a fresh problem."""
    desc, prim = W.get(1, 24)
    G = emx.Problem(desc)
    pd = G.upload_primaries(prim)
    kw = dict(n_slots=1 << 13, queue_capacity=1 << 18)
    a1 = G.transport(pd, 11, **kw)
    a2 = G.transport(pd, 11, **kw)                      # reused graph
    b = G.transport(pd, 12, **kw)                       # other seed
    a3 = G.transport(pd, 11, **kw)
    for x in (a2, a3):
        assert np.array_equal(x["steps"], a1["steps"]) and np.array_equal(x["inter"], a1["inter"])
        assert np.allclose(x["edep"], a1["edep"], rtol=1e-12)
    assert not np.array_equal(b["steps"], a1["steps"])
    fresh = emx.Problem(desc)
    f = fresh.transport(fresh.upload_primaries(prim), 12, **kw)
    assert np.array_equal(b["steps"], f["steps"]) and np.array_equal(b["inter"], f["inter"])
    prim2 = {k: v[:12].copy() for k, v in prim.items()}
    c = G.transport(G.upload_primaries(prim2), 11, **kw)            # other primaries
    f2 = fresh.transport(fresh.upload_primaries(prim2), 11, **kw)
    assert np.array_equal(c["steps"], f2["steps"]) and c["E_in"] == pytest.approx(a1["E_in"] / 2)
    d = G.transport(pd, 11, n_slots=1 << 12, queue_capacity=1 << 18)  # other workspace carve-up
    assert np.array_equal(d["steps"], a1["steps"])


def test_fringe_field_changes_the_result_and_uniform_limit_does_not(emx):
    """The fringe pushed out to |z| = 1e9 cm is the uniform field: same counters as config 4 (the stage-position
    integrator then does the same arithmetic); the real fringe of config 6 gives other histories."""
    d4, prim = W.get(4, 32)
    d6, _ = W.get(6, 32)
    far = dict(d6)
    far["field_fringe"] = (1e9, 1.0)
    kw = dict(n_slots=1 << 14, queue_capacity=1 << 20)
    res = []
    for desc in (d4, far, d6):
        G = emx.Problem(desc)
        res.append(G.transport(G.upload_primaries(prim), 4, **kw))
    assert np.array_equal(res[0]["steps"], res[1]["steps"]) and np.array_equal(res[0]["inter"], res[1]["inter"])
    assert np.allclose(res[0]["edep"], res[1]["edep"], rtol=1e-11, atol=1e-9)
    assert not np.array_equal(res[0]["steps"], res[2]["steps"])
    assert res[2]["edep"].sum() + res[2]["escaped"] + res[2]["looper"] == pytest.approx(res[2]["E_in"], rel=1e-9)


def test_error_paths(emx):
    import ctypes as C
    L = emx.lib()
    h = C.c_void_p()
    assert L.emx_create(C.byref(h)) == 0
    assert L.emx_set_field_fringe(h, 100.0, 15.0) == -1      # no field along z set
    assert L.emx_set_field(h, 0.0, 1.0, 0.0) == 0 and L.emx_set_field_fringe(h, 100.0, 15.0) == -1
    assert L.emx_set_field(h, 0.0, 0.0, 2.0) == 0 and L.emx_set_field_fringe(h, 100.0, -1.0) == -1
    assert L.emx_set_field_fringe(h, 100.0, 15.0) == 0
    assert L.emx_add_surface(h, 9, 1.0) == -1
    assert L.emx_build_tables(h, None) == -2           # no volume
    assert b"volume" in L.emx_last_error(h)
    assert L.emx_transport(h, 0, None, None, None, None, None, None, 0, 10, 10, None, 0, None) == -2
    hist = (C.c_uint64 * (3 * emx.NHIST))()
    assert L.emx_read_step_hist(h, C.cast(hist, C.c_void_p)) == -2      # no transport yet
    assert L.emx_read_step_hist(h, None) == -1
    L.emx_destroy(h)


def test_scheduling_knobs_do_not_change_results(emx):
    """Time slicing of the field propagation (attempts per iteration before a track may be parked), the grids of
    the persistent kernels, the shared-memory staging switches and the launch paths (the loop as one graph with a WHILE node, flat iteration graphs
    polled by the host, plain stream launches, profiled launches) only change WHEN work is done: counters are
    equal, tallies equal up to summation order."""
    desc, prim = W.get(4, 64)
    runs, hists = [], []
    variants = (dict(slice_min=2, slice_max=16), dict(slice_min=1000, slice_max=1000), dict(slice_min=1, slice_max=1),
                dict(slice_min=3, slice_max=7, profile=2), dict(profile=1), dict(loop_node=0),
                dict(blocks_per_sm={"k_field": 1, "k_a2": 2, "k_b<gamma>": 1}), dict(stage_faces=True, stage_tables=True))
    for v in variants:
        v = dict(v)
        G = emx.Problem(desc)
        G.set_profile(v.pop("profile", 0))
        G.set_schedule(slice_above=0, **v)
        runs.append(G.transport(G.upload_primaries(prim), desc["seed"], n_slots=1 << 14, queue_capacity=1 << 20))
        hists.append(G.read_step_hist())
    assert all(np.array_equal(hists[0], h) for h in hists[1:])
    a = runs[0]
    for b in runs[1:]:
        for k in ("steps", "tracks", "inter"):
            assert np.array_equal(a[k], b[k]), k
        assert a["null_int"] == b["null_int"]
        assert np.allclose(a["edep"], b["edep"], rtol=1e-11, atol=1e-9)
        assert b["escaped"] == pytest.approx(a["escaped"], rel=1e-11)
    assert runs[0]["iterations"] != runs[1]["iterations"] or runs[0]["iterations"] != runs[2]["iterations"]   # the schedules did differ


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 7])
def test_full_size_bench_configuration(emx, emo, cfg):
    """BASELINE configs 1, 2 and 3 in full (10 000 showers of 1 / 10 / 10 GeV) and config 4 in full (100 000 primaries, 2^20 slots, 2^26 records: what bench.py times), against
    the oracle on all host cores.  With keyed random numbers the histories are the same, so the integer
    counters agree to a few parts per million (a comparison within rounding of equality may flip in
    3.6e9 steps) and every tally within 1e-6; energy closes to 1e-9.  The same for config 7 in full (10 000
    showers of 10 GeV with multiple scattering and energy-loss fluctuations, 1.5e9 steps), as bench.py --config 7
    times it."""
    desc, prim = W.get(cfg)
    G = emx.Problem(desc)
    g = G.transport(G.upload_primaries(prim), desc["seed"])
    assert g["stalls"] == 0
    assert g["edep"].sum() + g["escaped"] + g["looper"] == pytest.approx(g["E_in"], rel=1e-9)
    assert g["track_steps"] == int(g["steps"].sum())
    o = emo.Problem(desc).transport(prim, desc["seed"])
    assert o["edep"].sum() + o["escaped"] + o["looper"] == pytest.approx(o["E_in"], rel=1e-9)
    for k in ("steps", "tracks", "inter"):
        a, b = o[k].astype(np.float64), g[k].astype(np.float64)
        assert np.all(np.abs(a - b) <= 1e-5 * np.maximum(a, 1.0) + 5.0), (k, o[k], g[k])
    big = o["edep"] > 1e-6 * o["E_in"]
    assert np.all(np.abs(g["edep"][big] - o["edep"][big]) <= 1e-6 * o["edep"][big])
    assert g["escaped"] == pytest.approx(o["escaped"], rel=1e-6)
    hg, ho = G.read_step_hist().astype(np.float64), o["step_hist"].astype(np.float64)
    assert hg.sum(1).tolist() == g["tracks"].astype(np.float64).tolist()
    assert np.all(np.abs(hg - ho) <= 1e-5 * ho + 5.0), np.abs(hg - ho).max()
