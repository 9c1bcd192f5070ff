"""ctypes binding of the ORACLE library (test infrastructure; see emo.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It imports nothing from paper_2203_09467_b200 except nothing at all: problem descriptions arrive as
plain dicts (the format produced by the workloads module, which holds no physics).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MAX_ELEM, MAX_FACES, NPROC, PER_PRIM, NHIST = 4, 8, 8, 11, 96
T_NAMES = ["compton", "photo", "pair", "moller", "brems_em", "dedx_em", "range_em", "bhabha", "brems_ep",
           "annih", "dedx_ep", "range_ep", "pair_elem0", "pair_elem1", "pair_elem2", "pair_elem3", "msc", "var_em", "var_ep", "msc2"]
T = {n: i for i, n in enumerate(T_NAMES)}
ME = 0.51099895000


class Physics(C.Structure):
    _fields_ = [("process_mask", C.c_uint), ("E_min", C.c_double), ("E_max", C.c_double), ("n_E", C.c_int),
                ("E_trk", C.c_double), ("prod_cut_cm", C.c_double), ("alpha_R", C.c_double), ("rho_R", C.c_double),
                ("lin_loss", C.c_double), ("field_eps", C.c_double), ("max_substeps", C.c_int),
                ("vacuum_step", C.c_double), ("max_steps", C.c_int), ("deposit_e_at_creation", C.c_int),
                ("msc", C.c_int), ("msc_fr", C.c_double), ("msc_smin", C.c_double), ("fluct", C.c_int),
                ("integrator", C.c_int)]


class Track(C.Structure):
    _fields_ = [("x", C.c_double * 3), ("u", C.c_double * 3), ("E", C.c_double), ("tid", C.c_uint64),
                ("prim", C.c_uint32), ("step", C.c_uint32), ("vol", C.c_int), ("surf", C.c_int),
                ("ptype", C.c_int), ("alive", C.c_int)]


class StepResult(C.Structure):
    _fields_ = [("trk", Track), ("action", C.c_int), ("process", C.c_int), ("n_sec", C.c_int),
                ("sec", Track * 4), ("sec_ord", C.c_int * 4), ("edep", C.c_double), ("edep_vol", C.c_int),
                ("below_cut", C.c_double), ("escaped", C.c_double), ("looper", C.c_double), ("s", C.c_double),
                ("msc_tau", C.c_double), ("n_draws", C.c_int), ("null_int", C.c_int), ("rest", C.c_int), ("n_sub", C.c_int)]


class Rng(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("prim", C.c_uint32), ("tid", C.c_uint64), ("step", C.c_uint32), ("n", C.c_uint32)]


class Scalars(C.Structure):
    _fields_ = [("escaped", C.c_double), ("below_cut", C.c_double), ("looper", C.c_double), ("E_in", C.c_double),
                ("steps", C.c_uint64 * 3), ("tracks", C.c_uint64 * 3), ("inter", C.c_uint64 * NPROC),
                ("null_int", C.c_uint64), ("track_steps", C.c_uint64), ("step_hist", (C.c_uint64 * NHIST) * 3)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        d, i, p = C.c_double, C.c_int, C.c_void_p
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        sig = {
            "emo_philox4x32_10": (None, [C.POINTER(C.c_uint32)] * 3),
            "emo_u01": (d, [C.c_uint32, C.c_uint32]),
            "emo_draw": (d, [C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint32, C.c_uint32]),
            "emo_child_tid": (C.c_uint64, [C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint32, C.c_uint32]),
            "emo_fc": (d, [i]), "emo_X0_elem_gcm2": (d, [i, d]), "emo_sigma_kn": (d, [d]),
            "emo_sigma_pe": (d, [i, d]), "emo_pair_dcs": (d, [i, d, d]), "emo_sigma_pair": (d, [i, d]),
            "emo_sigma_moller": (d, [d, d]), "emo_sigma_bhabha": (d, [d, d]), "emo_sigma_annih": (d, [d]),
            "emo_moller_dcs": (d, [d, d]), "emo_bhabha_dcs": (d, [d, d]),
            "emo_brems_Sigma": (d, [d, d, d]), "emo_brems_dedx": (d, [d, d, d]),
            "emo_gauss_legendre": (None, [i, dp, dp]),
            "emo_loss_second_moment": (d, [i, d, d]), "emo_fluctuate_loss": (d, [d, d, d, d, d]),
            "emo_msc_screening": (d, [i, d]), "emo_msc_sigma1": (d, [i, d, d]), "emo_msc_one_minus_mu": (d, [d, d]),
            "emo_msc_sigma2": (d, [i, d, d]), "emo_msc_phi3": (d, [d]), "emo_msc_geom_length": (d, [d, d]),
            "emo_msc_lateral_r2": (d, [d, d, d]),
            "emo_msc_deflect": (None, [C.POINTER(Rng), d, dp, dp]),
            "emo_create": (p, []), "emo_destroy": (None, [p]),
            "emo_add_material": (i, [p, i, ip, dp, dp, d, d]), "emo_add_surface": (i, [p, i, d]),
            "emo_add_volume": (i, [p, i, ip, ip, i, i]), "emo_set_field": (i, [p, d, d, d]), "emo_set_field_fringe": (i, [p, d, d]),
            "emo_field_profile": (None, [p, dp, dp]),
            "emo_rk4_doubling_map": (None, [p, dp, dp, d, d, dp, dp, dp]),
            "emo_dp45": (None, [p, dp, dp, d, d, dp, dp, dp]),
            "emo_set_physics": (i, [p, C.POINTER(Physics)]), "emo_set_cuts": (i, [p, i, d, d]),
            "emo_build_tables": (i, [p]), "emo_get_table": (i, [p, i, i, dp, i]),
            "emo_get_material_info": (i, [p, i, dp]), "emo_lookup": (d, [p, i, i, d]),
            "emo_range_inverse": (d, [p, i, i, d]),
            "emo_distance": (d, [p, i, dp, dp, i, ip]), "emo_neighbour": (i, [p, dp, dp, i]),
            "emo_locate": (i, [p, dp]),
            "emo_rk4_doubling": (None, [dp, dp, d, dp, d, dp, dp, dp]),
            "emo_propagate_field": (d, [p, i, ip, dp, dp, d, d, ip]),
            "emo_next": (d, [C.POINTER(Rng)]),
            "emo_rotate": (None, [dp, d, d, dp]),
            "emo_compton": (None, [C.POINTER(Rng), d, dp, dp, dp, dp, dp]),
            "emo_photo_dir": (None, [C.POINTER(Rng), d, dp, dp]),
            "emo_pair": (i, [C.POINTER(Rng), i, d, dp, dp, dp, dp, dp]),
            "emo_brems": (i, [C.POINTER(Rng), d, d, dp, dp, dp, dp, dp]),
            "emo_moller": (i, [C.POINTER(Rng), d, d, dp, dp, dp, dp, dp]),
            "emo_bhabha": (i, [C.POINTER(Rng), d, d, dp, dp, dp, dp, dp]),
            "emo_annih_flight": (None, [C.POINTER(Rng), d, dp, dp, dp, dp, dp]),
            "emo_annih_rest": (None, [C.POINTER(Rng), dp, dp]),
            "emo_step_bin": (i, [C.c_uint64]),
            "emo_step_batch": (i, [p, C.c_uint64, C.c_long, C.POINTER(Track), C.POINTER(StepResult)]),
            "emo_transport": (i, [p, C.c_long, ip, dp, dp, dp, ip, ip, C.c_uint64, i, dp, C.POINTER(Scalars), dp, dp]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def physics_from_dict(ph):
    s = Physics()
    for k, _ in Physics._fields_:
        setattr(s, k, ph[k])
    return s


class Problem:
    """Oracle problem built from a workload dict (materials, surfaces, volumes, field, physics)."""

    def __init__(self, desc):
        L = lib()
        self.desc = desc
        self.h = L.emo_create()
        for m in desc["materials"]:
            Z = np.asarray(m["Z"], dtype=np.int32)
            A = np.asarray(m["A"], dtype=np.float64)
            w = np.asarray(m["w"], dtype=np.float64)
            r = L.emo_add_material(self.h, len(Z), _ip(Z), _dp(A), _dp(w), m["rho"], m["I_eV"])
            assert r >= 0, "add_material"
        for (t, v) in desc["surfaces"]:
            assert L.emo_add_surface(self.h, int(t), float(v)) >= 0
        for vol in desc["volumes"]:
            s = np.asarray(vol["surf"], dtype=np.int32)
            e = np.asarray(vol["sense"], dtype=np.int32)
            assert L.emo_add_volume(self.h, len(s), _ip(s), _ip(e), vol["material"], vol["tally"]) >= 0
        B = desc.get("field", (0.0, 0.0, 0.0))
        L.emo_set_field(self.h, *[float(b) for b in B])
        if desc.get("field_fringe"):
            assert L.emo_set_field_fringe(self.h, *[float(v) for v in desc["field_fringe"]]) == 0
        ph = physics_from_dict(desc["physics"])
        assert L.emo_set_physics(self.h, C.byref(ph)) == 0
        for im, m in enumerate(desc["materials"]):
            if "Tcut" in m:
                L.emo_set_cuts(self.h, im, m["Tcut"], m["kcut"])
        assert L.emo_build_tables(self.h) == 0
        self.n_E = desc["physics"]["n_E"]
        self.n_tally = max([v["tally"] for v in desc["volumes"]] + [-1]) + 1

    def __del__(self):
        if getattr(self, "h", None):
            lib().emo_destroy(self.h)
            self.h = None

    def table(self, material, kind):
        out = np.empty(self.n_E)
        k = T[kind] if isinstance(kind, str) else kind
        assert lib().emo_get_table(self.h, material, k, _dp(out), self.n_E) == 0
        return out

    def material_info(self, material):
        o = np.empty(8)
        lib().emo_get_material_info(self.h, material, _dp(o))
        return dict(n_e=o[0], I=o[1], hwp=o[2], X0=o[3], Tcut=o[4], kcut=o[5], rho=o[6], n_elem=int(o[7]))

    def lookup(self, material, kind, E):
        return lib().emo_lookup(self.h, material, T[kind], float(E))

    def range_inverse(self, material, kind, r):
        return lib().emo_range_inverse(self.h, material, T[kind], float(r))

    def distance(self, vol, x, u, surf=-1):
        x = np.asarray(x, dtype=np.float64); u = np.asarray(u, dtype=np.float64)
        hit = C.c_int(-1)
        d = lib().emo_distance(self.h, vol, _dp(x), _dp(u), surf, C.byref(hit))
        return d, hit.value

    def neighbour(self, x, u, S):
        x = np.asarray(x, dtype=np.float64); u = np.asarray(u, dtype=np.float64)
        return lib().emo_neighbour(self.h, _dp(x), _dp(u), S)

    def locate(self, x):
        x = np.asarray(x, dtype=np.float64)
        return lib().emo_locate(self.h, _dp(x))

    def propagate_field(self, vol, surf, x, u, kappa, s_max):
        x = np.array(x, dtype=np.float64); u = np.array(u, dtype=np.float64)
        sf = C.c_int(surf); hit = C.c_int(-1)
        s = lib().emo_propagate_field(self.h, vol, C.byref(sf), _dp(x), _dp(u), kappa, s_max, C.byref(hit))
        return s, hit.value, x, u

    def step_batch(self, tracks, seed):
        """tracks: ctypes array of Track; returns ctypes array of StepResult."""
        n = len(tracks)
        out = (StepResult * n)()
        assert lib().emo_step_batch(self.h, seed, n, tracks, out) == 0
        return out

    def transport(self, prim, seed, n_threads=None, per_primary=False):
        """prim: dict with ptype (i32), E, pos (n,3), dir (n,3), vol (i32), surf (i32)."""
        n = len(prim["E"])
        n_threads = n_threads or (os.cpu_count() or 1)
        pt = np.ascontiguousarray(prim["ptype"], dtype=np.int32)
        E = np.ascontiguousarray(prim["E"], dtype=np.float64)
        pos = np.ascontiguousarray(prim["pos"], dtype=np.float64)
        dr = np.ascontiguousarray(prim["dir"], dtype=np.float64)
        vol = np.ascontiguousarray(prim["vol"], dtype=np.int32)
        srf = np.ascontiguousarray(prim["surf"], dtype=np.int32)
        edep = np.zeros(max(self.n_tally, 1))
        sc = Scalars()
        pp = np.zeros((n, PER_PRIM)) if per_primary else None
        ppt = np.zeros((n, max(self.n_tally, 1))) if per_primary else None
        r = lib().emo_transport(self.h, n, _ip(pt), _dp(E), _dp(pos), _dp(dr), _ip(vol), _ip(srf), seed, n_threads,
                                _dp(edep), C.byref(sc), _dp(pp) if per_primary else None,
                                _dp(ppt) if per_primary else None)
        assert r == 0, "emo_transport failed"
        res = dict(edep=edep[:self.n_tally], escaped=sc.escaped, below_cut=sc.below_cut, looper=sc.looper,
                   E_in=sc.E_in, steps=np.array(sc.steps[:], dtype=np.uint64),
                   tracks=np.array(sc.tracks[:], dtype=np.uint64), inter=np.array(sc.inter[:], dtype=np.uint64),
                   null_int=int(sc.null_int), track_steps=int(sc.track_steps),
                   step_hist=np.array([list(sc.step_hist[k]) for k in range(3)], dtype=np.uint64))
        if per_primary:
            res["per_prim"] = pp
            res["per_prim_tally"] = ppt[:, :self.n_tally]
        return res


def sample(kind, n, u=(0.0, 0.0, 1.0), seed=12345, **kw):
    """Run one of the samplers n times (each on its own keyed stream: prim = sample index).
    Returns a dict of arrays.  Test helper."""
    L = lib()
    u = np.asarray(u, dtype=np.float64)
    a = np.zeros(n); b = np.zeros(n); ok = np.ones(n, dtype=np.int32); nd = np.zeros(n, dtype=np.int32)
    v1 = np.zeros((n, 3)); v2 = np.zeros((n, 3))
    A, Bv = C.c_double(), C.c_double()
    w1 = np.zeros(3); w2 = np.zeros(3)
    for i in range(n):
        r = Rng(seed, i, 7, 3, 0)
        if kind == "compton":
            L.emo_compton(C.byref(r), kw["E"], _dp(u), C.byref(A), _dp(w1), C.byref(Bv), _dp(w2))
        elif kind == "photo":
            L.emo_photo_dir(C.byref(r), kw["E"], _dp(u), _dp(w1))
        elif kind == "pair":
            ok[i] = L.emo_pair(C.byref(r), kw["Z"], kw["E"], _dp(u), C.byref(A), _dp(w1), C.byref(Bv), _dp(w2))
        elif kind == "brems":
            ok[i] = L.emo_brems(C.byref(r), kw["T"], kw["kc"], _dp(u), C.byref(A), _dp(w1), C.byref(Bv), _dp(w2))
        elif kind == "moller":
            ok[i] = L.emo_moller(C.byref(r), kw["T"], kw["Tcut"], _dp(u), C.byref(A), _dp(w1), C.byref(Bv), _dp(w2))
        elif kind == "bhabha":
            ok[i] = L.emo_bhabha(C.byref(r), kw["T"], kw["Tcut"], _dp(u), C.byref(A), _dp(w1), C.byref(Bv), _dp(w2))
        elif kind == "annih":
            L.emo_annih_flight(C.byref(r), kw["T"], _dp(u), C.byref(A), _dp(w1), C.byref(Bv), _dp(w2))
        elif kind == "rest":
            L.emo_annih_rest(C.byref(r), _dp(w1), _dp(w2))
        else:
            raise ValueError(kind)
        a[i], b[i], nd[i] = A.value, Bv.value, r.n
        v1[i], v2[i] = w1, w2
    return dict(a=a, b=b, v1=v1, v2=v2, ok=ok, n_draws=nd)
