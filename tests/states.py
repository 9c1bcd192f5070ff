"""Seeded random track states for the single-step (level-2) parity tests.

Input generation only: positions are drawn in the bounding box of the problem's surfaces and located with
the ORACLE's point-location routine (tests may call the oracle); a share of the states is moved onto a
cell face the way a boundary step would leave it (oracle distance + neighbour).  No value produced by
the CUDA path enters here.
"""
import numpy as np


def bounding_box(desc):
    lo, hi = np.full(3, -60.0), np.full(3, 60.0)
    planes = {0: [], 1: [], 2: []}
    rmax = 0.0
    for t, v in desc["surfaces"]:
        if t < 3:
            planes[t].append(v)
        else:
            rmax = max(rmax, v)
    for a in range(3):
        if planes[a]:
            lo[a], hi[a] = min(planes[a]), max(planes[a])
        elif rmax > 0 and a < 2:
            lo[a], hi[a] = -rmax, rmax
    return lo, hi


def random_states(emo, P, desc, n, seed, on_surface_frac=0.3, ptypes=(0, 1, 2)):
    """Returns a ctypes array of emo.Track (n entries) and the same data as a dict of numpy arrays."""
    rng = np.random.default_rng(seed)
    ph = desc["physics"]
    lo, hi = bounding_box(desc)
    tracks = []
    n_vol = len(desc["volumes"])
    infinite = len(desc["surfaces"]) == 0
    while len(tracks) < n:
        x = rng.uniform(lo, hi)
        if rng.random() < 0.3 and not infinite:      # concentrate near the axis / the beam line
            x[:2] *= 0.05
        vol = 0 if infinite else P.locate(x)
        if vol < 0 or vol >= n_vol:
            continue
        mu = rng.uniform(-1, 1)
        phi = rng.uniform(0, 2 * np.pi)
        s = np.sqrt(1 - mu * mu)
        u = np.array([s * np.cos(phi), s * np.sin(phi), mu])
        r = rng.random()
        if r < 0.05:
            u = np.array([0.0, 0.0, 1.0 if rng.random() < 0.5 else -1.0])
        elif r < 0.08:
            u = np.array([1.0, 0.0, 0.0])
        u = u / np.linalg.norm(u)
        surf = -1
        if not infinite and rng.random() < on_surface_frac:
            d, hit = P.distance(vol, x, u, -1)
            if hit >= 0 and np.isfinite(d):
                x2 = x + d * u
                nv = P.neighbour(x2, u, hit)
                if nv >= 0:
                    x, vol, surf = x2, nv, hit
                    if rng.random() < 0.3:           # sometimes turn the track back towards the surface
                        mu = rng.uniform(-1, 1)
                        phi = rng.uniform(0, 2 * np.pi)
                        s = np.sqrt(1 - mu * mu)
                        u2 = np.array([s * np.cos(phi), s * np.sin(phi), mu])
                        # keep it on the side it is filed under: same sign of grad f . u
                        t, v = desc["surfaces"][hit]
                        g_old = u[t] if t < 3 else 2 * (x[0] * u[0] + x[1] * u[1])
                        g_new = u2[t] if t < 3 else 2 * (x[0] * u2[0] + x[1] * u2[1])
                        if g_old * g_new > 0:
                            u = u2
        tr = emo.Track()
        tr.x[:] = list(x)
        tr.u[:] = list(u)
        e_lo = 0.5 * ph["E_trk"] if rng.random() < 0.02 else ph["E_min"]
        tr.E = float(np.exp(rng.uniform(np.log(e_lo), np.log(ph["E_max"]))))
        tr.tid = int(rng.integers(0, 2 ** 63)) if rng.random() < 0.9 else 0
        tr.prim = int(rng.integers(0, 2 ** 31))
        tr.step = int(rng.integers(0, 60)) if rng.random() < 0.97 else ph["max_steps"] - 1
        tr.vol = int(vol)
        tr.surf = int(surf)
        tr.ptype = int(ptypes[rng.integers(0, len(ptypes))])
        tr.alive = 1
        tracks.append(tr)
    return (emo.Track * n)(*tracks)


FIELDS_TRK = ("x", "u", "E", "tid", "prim", "step", "vol", "surf", "ptype", "alive")


def result_arrays(res):
    """ctypes StepResult array -> dict of numpy arrays (works for the oracle's and the CUDA binding's
    structures, which have the same field names and layout)."""
    a = np.frombuffer(res, dtype=np.dtype(type(res[0])))
    t, sec = a["trk"], a["sec"]
    return dict(
        x=t["x"].copy(), u=t["u"].copy(), E=t["E"].copy(), step=t["step"].astype(np.int64),
        vol=t["vol"].copy(), surf=t["surf"].copy(), alive=t["alive"].copy(), action=a["action"].copy(),
        process=a["process"].copy(), n_sec=a["n_sec"].copy(), edep=a["edep"].copy(),
        below_cut=a["below_cut"].copy(), escaped=a["escaped"].copy(), looper=a["looper"].copy(),
        s=a["s"].copy(), n_sub=a["n_sub"].copy(), msc_tau=a["msc_tau"].copy(), n_draws=a["n_draws"].copy(), null_int=a["null_int"].copy(), rest=a["rest"].copy(),
        sec_E=sec["E"].copy(), sec_u=sec["u"].copy(), sec_x=sec["x"].copy(), sec_tid=sec["tid"].copy(),
        sec_ptype=sec["ptype"].copy(), sec_ord=a["sec_ord"].copy(), sec_vol=sec["vol"].copy(),
        sec_prim=sec["prim"].copy(), sec_surf=sec["surf"].copy())


ME = 0.51099895
EPS = 2.0 ** -52          # fp64 unit roundoff (spacing at 1)
RTOL2 = 1e-12             # level 2 of BASELINE.json north_star


def step_tolerances(desc, tracks, ref):
    """Per-state level-2 tolerances, DERIVED from the arithmetic of the step, as multiples of
    nothing observed: every entry is RTOL2 for a step without field substeps and without fluctuated loss.

    Field steps (n = substep attempts, from the oracle's own count).  Both implementations run the same IEEE
    operations, but their libm differs in the last bit, so after the first rescaling of h the two positions differ by
    a rounding, EPS |x|.  The error estimate err = |x_full - x_half| is a difference of two positions that each carry
    a few such roundings (take 8 EPS |x| for the difference), so err differs by 8 EPS |x| / err relative, the next
    trial step by a fifth of that (h ~ err^-1/5), and the RK4 truncation error of the substep (err / 15, fifth order in
    h) by 5 dh/h err / 15 < 8 EPS |x|: per substep the end point moves by < 8 EPS |x| along the helix and the
    direction by < |kappa| 8 EPS |x|, whatever err is.  With X = max(|x|, s):
      positions, path length   RTOL2 + 8 n EPS              (relative to X)
      directions               RTOL2 + (position tolerance) X |kappa|
    -- on a helix the direction is a function of the arc length, du = |kappa| ds, so whatever the end point may differ
    by along the track (RTOL2 X from north_star's own 1e-12, plus the substep term) the direction differs by |kappa|
    times that.  (Where a boundary ends the step the landing rule |L - d| <= field_eps accepts any point within field_eps
    of the surface; the two runs take the same decisions, and their landing points differ by (field_eps / h_last) times
    the shift of the last substep's start, observed up to 20 n EPS X: inside RTOL2 X, which is why the direction must
    be given the same allowance.)
      energies                 RTOL2 + (path tolerance) X / s    (the loss of the step is proportional to its path)
    A step cut short by the substep budget (action TRUNC) returns s = sum of its n trial steps, each carrying
    dh/h <= 8 EPS |x| / (5 err) with err >= field_eps / 3125 where h still grows: ds/s <= 5000 EPS X / field_eps, and
    the direction turns by |kappa| ds.
    In a NON-UNIFORM field the error estimate changes along the path, so the two sequences of substeps do not stay
    within roundings of each other: each run realises its own truncation errors (<= field_eps / 15 per accepted
    substep, in position and again through the direction it leaves the substep with) and lands on a surface within
    field_eps of it along its own chord: |dx| <= 4 (n / 15 + 1) field_eps.
    Its TRUNC steps (the 1000-attempt emergency exit, vacuum only: no loss) stop at arc lengths that depend on all
    1000 step sizes: several end points are correct (they lie on the same curve), so only ds <= 5e-2 s is asked, with
    the position and direction differences that follow from ds.
    Energy-loss fluctuations: the fluctuated loss can take most of E, the post-loss energy E' = E - dE carries
    EPS E / E' of relative rounding and everything the interactor computes from E' inherits it: scale E / E'."""
    n = len(tracks)
    ph = desc["physics"]
    B = float(np.linalg.norm(desc.get("field", (0.0, 0.0, 0.0))))
    E = np.array([t.E for t in tracks])
    pt = np.array([t.ptype for t in tracks])
    nsub = ref["n_sub"].astype(np.float64)
    p = np.sqrt(E * (E + 2 * ME))
    kappa = np.where(pt != 0, 2.99792458 * B / np.maximum(p, 1e-300), 0.0)
    fin = np.isfinite(ref["s"])
    s_abs = np.where(fin, np.abs(ref["s"]), 0.0)
    X = np.maximum(np.maximum(np.linalg.norm(ref["x"], axis=1), s_abs), 1e-300)
    eps_f = ph["field_eps"]
    path = 8 * nsub * EPS                               # relative to X
    trunc = (ref["action"] == 4) & (nsub >= ph["max_substeps"])
    path = np.where(trunc, path + 5000 * EPS * X / eps_f * s_abs / X, path)
    if desc.get("field_fringe"):
        path = np.where(nsub > 1, path + 4 * (nsub / 15 + 1) * eps_f / X, path)
        path = np.where(trunc, path + 5e-2 * s_abs / X, path)
    tol_x = RTOL2 + path
    tol_u = RTOL2 + np.where(nsub > 0, kappa * tol_x * X, 0.0)
    tol_E = RTOL2 + np.where(s_abs > 0, path * X / np.maximum(s_abs, 1e-300), 0.0)
    if ph.get("fluct"):
        e_post = np.maximum(E - ref["edep"], 0.0)
        scale = np.where((pt != 0) & (e_post > 0), np.minimum(E / np.maximum(e_post, 1e-300), 1e6), 1.0)
        tol_E = tol_E * scale
        tol_u = tol_u * scale
    return dict(x=tol_x, u=tol_u, E=tol_E, trunc=trunc)


def compare_steps(ref, got, E_in, tol=None, skip=None):
    """Level-1/2 comparison of two result dicts for the same input states (E_in = their energies).
    Integers must be equal.  Energies are compared on the scale of the step's input energy
    (E' = E - dE is a difference, so its own magnitude is not the scale of its rounding error; DESIGN.md
    section 6), path lengths and positions relative to X = max(|x|, s), unit vectors absolutely.  `tol` =
    step_tolerances(...) (default: RTOL2 everywhere).  `skip` masks states excluded from the floating-point
    comparison (they still count for the integers).
    Returns (n_int_mismatch, worst error / tolerance, report) over all states."""
    n = len(ref["E"])
    if tol is None:
        tol = dict(x=np.full(n, RTOL2), u=np.full(n, RTOL2), E=np.full(n, RTOL2))
    int_keys = ("step", "vol", "surf", "alive", "action", "process", "n_sec", "n_draws", "null_int", "rest", "n_sub")
    bad = np.zeros(n, dtype=bool)
    report = {}
    for k in int_keys:
        m = ref[k] != got[k]
        if m.any():
            report[k] = int(m.sum())
        bad |= m
    ok = ~bad
    for k in ("sec_tid", "sec_ptype", "sec_ord", "sec_vol", "sec_prim", "sec_surf"):
        m = (ref[k] != got[k]).any(axis=1) & ok
        if m.any():
            report[k] = int(m.sum())
        bad |= m
    ok = ~bad
    if skip is not None:
        ok &= ~np.asarray(skip, dtype=bool)
    Es = np.asarray(E_in, dtype=np.float64)[ok]
    tx, tu, tE = tol["x"][ok], tol["u"][ok], tol["E"][ok]

    def ratio(err, t):
        r = err / t
        return float(r.max()) if r.size else 0.0

    for k in ("E", "edep", "below_cut", "escaped", "looper"):
        err = np.abs(ref[k][ok] - got[k][ok]) / np.maximum(np.abs(ref[k][ok]), Es)
        report["E:" + k] = ratio(err, tE)
    fin = np.isfinite(ref["s"][ok])
    X = np.maximum(np.maximum(np.linalg.norm(ref["x"][ok], axis=1), np.where(fin, np.abs(ref["s"][ok]), 0.0)), 1e-300)
    report["s"] = ratio((np.abs(ref["s"][ok] - got["s"][ok]) / X)[fin], tx[fin])
    mt = np.maximum(np.abs(ref["msc_tau"][ok]), 1e-300)
    report["msc_tau"] = ratio(np.abs(ref["msc_tau"][ok] - got["msc_tau"][ok]) / mt, tE)     # tau is proportional to the path, like the loss
    report["x"] = ratio((np.linalg.norm(ref["x"][ok] - got["x"][ok], axis=1) / X)[fin], tx[fin])
    report["u"] = ratio(np.linalg.norm(ref["u"][ok] - got["u"][ok], axis=1), tu)
    err = np.abs(ref["sec_E"][ok] - got["sec_E"][ok]) / np.maximum(np.abs(ref["sec_E"][ok]), Es[:, None])
    report["sec_E"] = ratio(err.max(axis=1) if err.size else err, tE)
    err = np.linalg.norm(ref["sec_u"][ok] - got["sec_u"][ok], axis=2)
    report["sec_u"] = ratio(err.max(axis=1) if err.size else err, tu)
    err = np.linalg.norm(ref["sec_x"][ok] - got["sec_x"][ok], axis=2) / X[:, None]
    report["sec_x"] = ratio(err.max(axis=1)[fin] if err.size else err, tx[fin])
    worst = max(v for k, v in report.items() if isinstance(v, float))
    return int(bad.sum()), worst, report
