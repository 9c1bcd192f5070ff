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


def compare_steps(ref, got, E_in, skip=None):
    """Level-1/2 comparison of two result dicts for the same input states (E_in = their energies).
    Integers must be equal.  Energies are compared on the scale of the step's input energy
    (E' = E - dE is a difference, so its own magnitude is not the scale of its rounding error; DESIGN.md
    section 6), lengths relative to themselves, positions relative to max(|x|, s), unit vectors absolutely.
    Directions are divided by 1 + 2e-3 gamma (gamma = E_in / me): emission angles are ~1/gamma and are
    formed from 1 - mu, so their rounding error is ~ eps_mach gamma.  `skip` masks states excluded from the
    floating-point comparison (they still count for the integers).
    Returns (n_int_mismatch, worst_rel, report) over all states."""
    n = len(ref["E"])
    int_keys = ("step", "vol", "surf", "alive", "action", "process", "n_sec", "n_draws", "null_int", "rest")
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
    worst = 0.0
    tiny = 1e-300

    def rel(a, b, scale=None):
        sc = np.maximum(np.abs(a), tiny) if scale is None else scale
        return np.abs(a - b) / sc

    ok = ~bad
    if skip is not None:
        ok &= ~np.asarray(skip, dtype=bool)
    Es = np.asarray(E_in, dtype=np.float64)[ok]
    cond = 1.0 + 2e-3 * Es / ME
    for k in ("E", "edep", "below_cut", "escaped", "looper"):
        r = rel(ref[k][ok], got[k][ok], np.maximum(np.abs(ref[k][ok]), Es))
        w = float(r.max()) if r.size else 0.0
        report["rel_" + k] = w
        worst = max(worst, w)
    fin = np.isfinite(ref["s"][ok])
    r = rel(ref["s"][ok][fin], got["s"][ok][fin])
    report["rel_s"] = float(r.max()) if r.size else 0.0
    r = rel(ref["msc_tau"][ok][fin], got["msc_tau"][ok][fin])
    report["rel_msc_tau"] = float(r.max()) if r.size else 0.0
    xs = np.maximum(np.linalg.norm(ref["x"][ok], axis=1), np.where(fin, np.abs(ref["s"][ok]), 0.0))
    d = np.linalg.norm(ref["x"][ok] - got["x"][ok], axis=1)
    d = d[fin] / np.maximum(xs[fin], 1e-30)
    report["rel_x"] = float(d.max()) if d.size else 0.0
    d = np.linalg.norm(ref["u"][ok] - got["u"][ok], axis=1) / cond
    report["abs_u"] = float(d.max()) if d.size else 0.0
    r = rel(ref["sec_E"][ok], got["sec_E"][ok], np.maximum(np.abs(ref["sec_E"][ok]), Es[:, None]))
    report["rel_sec_E"] = float(r.max()) if r.size else 0.0
    d = np.linalg.norm(ref["sec_u"][ok] - got["sec_u"][ok], axis=2) / cond[:, None]
    report["abs_sec_u"] = float(d.max()) if d.size else 0.0
    d = np.linalg.norm(ref["sec_x"][ok] - got["sec_x"][ok], axis=2)
    d = d[fin] / np.maximum(xs[fin], 1e-30)[:, None]
    report["rel_sec_x"] = float(d.max()) if d.size else 0.0
    worst = max(report[k] for k in report if k.startswith("rel_") or k.startswith("abs_"))
    return int(bad.sum()), worst, report
