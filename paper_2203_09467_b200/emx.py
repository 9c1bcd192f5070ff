"""Thin Python binding of the C-ABI in include/emx.h (same names; argument marshalling only).

PyTorch provides device memory and the CUDA stream; every step of the path runs in the kernels of
libemx.so.  There is no CPU fallback: if the library is missing or no CUDA device is present the calls
raise.  Problem descriptions are the plain dicts produced by `workloads` (inputs only).
"""
import atexit
import ctypes as C
import os
import weakref

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libemx.so")
MAX_ELEM, MAX_FACES, NPROC, NTABLE, NHIST = 4, 8, 8, 20, 96
# the step kernels in the order of emx_get_profile / emx_get_lanes / emx_schedule.blocks_per_sm
STAGES = ["k_a<gamma>", "k_a<charged>", "k_a0", "k_field", "k_a2", "k_b<gamma>", "k_b<charged>"]
T_NAMES = ["compton", "photo", "pair", "moller", "brems_em", "dedx_em", "range_em", "bhabha", "brems_ep",
           "annih", "dedx_ep", "range_ep", "pair_elem0", "pair_elem1", "pair_elem2", "pair_elem3", "msc", "var_em", "var_ep", "msc2"]
T = {n: i for i, n in enumerate(T_NAMES)}


class Physics(C.Structure):
    _fields_ = [("process_mask", C.c_uint32), ("E_min", C.c_double), ("E_max", C.c_double), ("n_E", C.c_int32),
                ("E_trk", C.c_double), ("prod_cut_cm", C.c_double), ("alpha_R", C.c_double), ("rho_R", C.c_double),
                ("lin_loss", C.c_double), ("field_eps", C.c_double), ("max_substeps", C.c_int32),
                ("vacuum_step", C.c_double), ("max_steps", C.c_int32), ("deposit_e_at_creation", C.c_int32),
                ("msc", C.c_int32), ("msc_fr", C.c_double), ("msc_smin", C.c_double), ("fluct", C.c_int32),
                ("integrator", C.c_int32)]


class Scalars(C.Structure):
    _fields_ = [("escaped", C.c_double), ("below_cut", C.c_double), ("looper", C.c_double), ("E_in", C.c_double),
                ("steps", C.c_uint64 * 3), ("tracks", C.c_uint64 * 3), ("inter", C.c_uint64 * NPROC),
                ("null_int", C.c_uint64), ("track_steps", C.c_uint64), ("stalls", C.c_uint64),
                ("iterations", C.c_uint64), ("peak_live", C.c_uint64), ("peak_queue", C.c_uint64)]


class Schedule(C.Structure):
    _fields_ = [("loop_node", C.c_int32), ("slice_min", C.c_int32), ("slice_max", C.c_int32), ("slice_above", C.c_int64),
                ("blocks_per_sm", C.c_int32 * 8), ("admit_below", C.c_int64), ("mev_per_slot", C.c_int32), ("reserved", C.c_int32)]


class Track(C.Structure):
    _fields_ = [("x", C.c_double * 3), ("u", C.c_double * 3), ("E", C.c_double), ("tid", C.c_uint64),
                ("prim", C.c_uint32), ("step", C.c_uint32), ("vol", C.c_int32), ("surf", C.c_int32),
                ("ptype", C.c_int32), ("alive", C.c_int32)]


class StepResult(C.Structure):
    _fields_ = [("trk", Track), ("action", C.c_int32), ("process", C.c_int32), ("n_sec", C.c_int32),
                ("sec", Track * 4), ("sec_ord", C.c_int32 * 4), ("edep", C.c_double), ("edep_vol", C.c_int32),
                ("below_cut", C.c_double), ("escaped", C.c_double), ("looper", C.c_double), ("s", C.c_double),
                ("msc_tau", C.c_double), ("n_draws", C.c_int32), ("null_int", C.c_int32), ("rest", C.c_int32),
                ("n_sub", C.c_int32)]


EXPORTS = ["emx_create", "emx_destroy", "emx_add_material", "emx_add_surface", "emx_add_volume", "emx_set_field", "emx_set_field_fringe",
           "emx_get_physics", "emx_set_physics", "emx_set_cuts", "emx_build_tables", "emx_get_table",
           "emx_get_material_info", "emx_n_tally", "emx_workspace_bytes", "emx_transport", "emx_transport_host",
           "emx_staging_bytes", "emx_set_primary_offset", "emx_get_schedule", "emx_set_schedule", "emx_neighbour_candidates", "emx_reset_tallies", "emx_read_tallies", "emx_read_step_hist", "emx_last_transport_ms", "emx_set_profile", "emx_get_profile", "emx_get_lanes",
           "emx_get_iteration_log", "emx_get_iteration_times",
           "emx_step_batch", "emx_field_substep_batch", "emx_philox_batch", "emx_draw_batch", "emx_refill_plan", "emx_refill_plan_static", "emx_refill_plan_static_max",
           "emx_refill_plan_static_setup", "emx_last_error",
           "emx_version"]

_lib = None


def lib():
    """Loads libemx.so (built in-tree by `python -m paper_2203_09467_b200.build`).  Raises if missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libemx.so not built: run `python -m paper_2203_09467_b200.build` (needs nvcc); "
                               "this package has no CPU path")
        import torch  # noqa: F401  -- load torch's CUDA libraries before ours (device memory and streams are torch's)
        L = C.CDLL(LIB_PATH)
        vp, i, l, d, u64 = C.c_void_p, C.c_int, C.c_long, C.c_double, C.c_uint64
        sig = {
            "emx_create": (i, [C.POINTER(vp)]), "emx_destroy": (None, [vp]),
            "emx_add_material": (i, [vp, i, vp, vp, vp, d, d]), "emx_add_surface": (i, [vp, i, d]),
            "emx_add_volume": (i, [vp, i, vp, vp, i, i]), "emx_set_field": (i, [vp, d, d, d]), "emx_set_field_fringe": (i, [vp, d, d]),
            "emx_get_physics": (i, [vp, C.POINTER(Physics)]), "emx_set_physics": (i, [vp, C.POINTER(Physics)]),
            "emx_set_cuts": (i, [vp, i, d, d]), "emx_build_tables": (i, [vp, vp]),
            "emx_get_table": (i, [vp, i, i, vp, i]), "emx_get_material_info": (i, [vp, i, vp]),
            "emx_n_tally": (i, [vp]), "emx_workspace_bytes": (C.c_size_t, [vp, l, l]),
            "emx_transport": (i, [vp, l, vp, vp, vp, vp, vp, vp, u64, l, l, vp, C.c_size_t, vp]),
            "emx_transport_host": (i, [vp, l, vp, vp, vp, vp, vp, vp, u64, l, l, vp, C.c_size_t, vp]),
            "emx_reset_tallies": (i, [vp, vp]), "emx_read_tallies": (i, [vp, vp, C.POINTER(Scalars)]),
            "emx_last_transport_ms": (d, [vp]), "emx_get_iteration_log": (l, [vp, vp, l]),
            "emx_get_iteration_times": (l, [vp, vp, l]),
            "emx_get_lanes": (i, [vp, vp]), "emx_read_step_hist": (i, [vp, vp]), "emx_set_primary_offset": (i, [vp, l]), "emx_staging_bytes": (C.c_size_t, [l]),
            "emx_get_schedule": (i, [vp, C.POINTER(Schedule)]), "emx_set_schedule": (i, [vp, C.POINTER(Schedule)]), "emx_neighbour_candidates": (i, [vp, i, i, i, vp, i]),
            "emx_set_profile": (i, [vp, i]), "emx_get_profile": (i, [vp, vp, vp, vp]),
            "emx_step_batch": (i, [vp, u64, l, vp, vp, vp]),
            "emx_philox_batch": (i, [l, vp, vp, vp, vp]),
            "emx_draw_batch": (i, [u64, l, vp, vp, vp, vp, vp, vp, vp]),
            "emx_refill_plan": (i, [l, l, l, vp, vp, vp, vp]),
            "emx_field_substep_batch": (i, [vp, l, vp, vp, vp, vp, vp, vp, vp, vp]),
            "emx_refill_plan_static": (i, [l, l, l, vp, vp, vp, vp]),
            "emx_refill_plan_static_max": (l, []), "emx_refill_plan_static_setup": (i, []),
            "emx_last_error": (C.c_char_p, [vp]), "emx_version": (C.c_char_p, []),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: the emx path runs on the GPU only (no CPU fallback)")
    return torch


def _stream():
    return C.c_void_p(_torch().cuda.current_stream().cuda_stream)


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _hp(a):
    return a.ctypes.data_as(C.c_void_p)


class EmxError(RuntimeError):
    pass


_live = weakref.WeakSet()


@atexit.register
def _destroy_all():
    """Free every problem while the CUDA runtime is still up (not from __del__ at interpreter teardown)."""
    for p in list(_live):
        p.close()


class Problem:
    """create -> add materials / surfaces / volumes -> set field / physics -> build tables."""

    def __init__(self, desc, build=True):
        L = lib()
        h = C.c_void_p()
        self._check(L.emx_create(C.byref(h)), None)
        self.h = h
        self._destroy = L.emx_destroy
        _live.add(self)
        self.desc = desc
        for m in desc["materials"]:
            Z, A, w = _np(m["Z"], np.int32), _np(m["A"], np.float64), _np(m["w"], np.float64)
            self._check(L.emx_add_material(h, len(Z), _hp(Z), _hp(A), _hp(w), m["rho"], m["I_eV"]))
        for (t, v) in desc["surfaces"]:
            self._check(L.emx_add_surface(h, int(t), float(v)))
        for vol in desc["volumes"]:
            s, e = _np(vol["surf"], np.int32), _np(vol["sense"], np.int32)
            self._check(L.emx_add_volume(h, len(s), _hp(s), _hp(e), vol["material"], vol["tally"]))
        B = desc.get("field", (0.0, 0.0, 0.0))
        self._check(L.emx_set_field(h, float(B[0]), float(B[1]), float(B[2])))
        if desc.get("field_fringe"):
            self._check(L.emx_set_field_fringe(h, float(desc["field_fringe"][0]), float(desc["field_fringe"][1])))
        ph = Physics()
        for k, _ in Physics._fields_:
            setattr(ph, k, desc["physics"][k])
        self._check(L.emx_set_physics(h, C.byref(ph)))
        for im, m in enumerate(desc["materials"]):
            if "Tcut" in m:
                self._check(L.emx_set_cuts(h, im, m["Tcut"], m["kcut"]))
        self.n_E = desc["physics"]["n_E"]
        self.n_tally = L.emx_n_tally(h)
        self._ws = None
        if build:
            self.build_tables()

    def _check(self, rc, h="self"):
        if rc < 0:
            hh = self.h if h == "self" else None
            raise EmxError("emx error %d: %s" % (rc, (lib().emx_last_error(hh) or b"").decode()))
        return rc

    def close(self):
        h, self.h = getattr(self, "h", None), None
        if h:
            self._ws = None
            self._destroy(h)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def build_tables(self):
        _torch()
        self._check(lib().emx_build_tables(self.h, _stream()))

    def table(self, material, kind):
        out = np.empty(self.n_E)
        self._check(lib().emx_get_table(self.h, material, T[kind] if isinstance(kind, str) else kind, _hp(out), self.n_E))
        return out

    def material_info(self, material):
        o = np.empty(8)
        self._check(lib().emx_get_material_info(self.h, material, _hp(o)))
        return dict(n_e=o[0], I=o[1], hwp=o[2], X0=o[3], Tcut=o[4], kcut=o[5], rho=o[6], n_elem=int(o[7]))

    def workspace(self, n_slots, queue_capacity, n_staged=0):
        """A torch uint8 CUDA tensor of emx_workspace_bytes() (+ emx_staging_bytes(n_staged) for
        emx_transport_host); cached per (n_slots, queue_capacity) and grown when more staging is asked for."""
        torch = _torch()
        key = (int(n_slots), int(queue_capacity))
        nb = lib().emx_workspace_bytes(self.h, key[0], key[1])
        if nb == 0:
            raise EmxError("emx_workspace_bytes: invalid sizes")
        nb += lib().emx_staging_bytes(int(n_staged)) if n_staged else 0
        if self._ws is None or self._ws[0] != key or self._ws[1].numel() < nb:
            self._ws = None
            self._ws = (key, torch.empty(nb, dtype=torch.uint8, device="cuda"))
        return self._ws[1]

    def upload_primaries(self, prim):
        """dict of numpy arrays -> dict of CUDA tensors (ptype i32, E, pos (n,3), dir (n,3), vol, surf)."""
        torch = _torch()
        dt = dict(ptype=np.int32, E=np.float64, pos=np.float64, dir=np.float64, vol=np.int32, surf=np.int32)
        return {k: torch.from_numpy(np.array(prim[k], dtype=dt[k], order="C")).cuda() for k in dt}

    def transport(self, prim_dev, seed, n_slots=None, queue_capacity=None, reset=True):
        """emx_transport on device-resident primaries.  Returns the tallies dict."""
        L = lib()
        n_slots = n_slots or self.desc["n_slots"]
        queue_capacity = queue_capacity or self.desc["queue_capacity"]
        ws = self.workspace(n_slots, queue_capacity)
        st = _stream()
        if reset:
            self._check(L.emx_reset_tallies(self.h, st))
        n = int(prim_dev["E"].numel())
        p = lambda k: C.c_void_p(prim_dev[k].data_ptr())
        self._check(L.emx_transport(self.h, n, p("ptype"), p("E"), p("pos"), p("dir"), p("vol"), p("surf"), seed,
                                    n_slots, queue_capacity, C.c_void_p(ws.data_ptr()), ws.numel(), st))
        return self.read_tallies()

    def transport_host(self, prim, seed, n_slots=None, queue_capacity=None, reset=True):
        """emx_transport_host: primaries in host memory (numpy), copies inside the call."""
        L = lib()
        n_slots = n_slots or self.desc["n_slots"]
        queue_capacity = queue_capacity or self.desc["queue_capacity"]
        ws = self.workspace(n_slots, queue_capacity, n_staged=len(prim["E"]))
        st = _stream()
        if reset:
            self._check(L.emx_reset_tallies(self.h, st))
        a = dict(ptype=_np(prim["ptype"], np.int32), E=_np(prim["E"], np.float64), pos=_np(prim["pos"], np.float64),
                 dir=_np(prim["dir"], np.float64), vol=_np(prim["vol"], np.int32), surf=_np(prim["surf"], np.int32))
        self._check(L.emx_transport_host(self.h, len(a["E"]), _hp(a["ptype"]), _hp(a["E"]), _hp(a["pos"]), _hp(a["dir"]),
                                         _hp(a["vol"]), _hp(a["surf"]), seed, n_slots, queue_capacity,
                                         C.c_void_p(ws.data_ptr()), ws.numel(), st))
        return self.read_tallies()

    def read_tallies(self):
        edep = np.zeros(max(self.n_tally, 1))
        sc = Scalars()
        self._check(lib().emx_read_tallies(self.h, _hp(edep), C.byref(sc)))
        return dict(edep=edep[:self.n_tally], escaped=sc.escaped, below_cut=sc.below_cut, looper=sc.looper,
                    E_in=sc.E_in, steps=np.array(sc.steps[:], dtype=np.uint64),
                    tracks=np.array(sc.tracks[:], dtype=np.uint64), inter=np.array(sc.inter[:], dtype=np.uint64),
                    null_int=int(sc.null_int), track_steps=int(sc.track_steps), stalls=int(sc.stalls),
                    iterations=int(sc.iterations), peak_live=int(sc.peak_live), peak_queue=int(sc.peak_queue),
                    ms=lib().emx_last_transport_ms(self.h))

    def neighbour_candidates(self, surface, sense, which):
        """cells tested, in order, after crossing `surface` towards `sense` (which = 0: listing it, 1: not listing it)"""
        n = lib().emx_neighbour_candidates(self.h, int(surface), int(sense), int(which), None, 0)
        if n < 0:
            self._check(n)
        out = np.zeros(max(n, 1), dtype=np.int32)
        lib().emx_neighbour_candidates(self.h, int(surface), int(sense), int(which), out.ctypes.data, n)
        return out[:n]

    def set_primary_offset(self, first):
        """the primaries of the following transports are primaries first, first + 1, ... of a longer list"""
        self._check(lib().emx_set_primary_offset(self.h, int(first)))

    def read_step_hist(self):
        """(3, NHIST) uint64: tracks of the last transport by particle type and steps-per-track bin"""
        h = np.zeros((3, NHIST), dtype=np.uint64)
        self._check(lib().emx_read_step_hist(self.h, _hp(h)))
        return h

    def set_schedule(self, **kw):
        """emx_set_schedule: loop_node, slice_min, slice_max, slice_above, blocks_per_sm (dict stage name -> blocks
        or a list of 7), stage_faces / stage_tables (bool: the shared-memory staging switches, both measured slower).  Only what is named changes.  A schedule never changes a result."""
        sc = Schedule()
        self._check(lib().emx_get_schedule(self.h, C.byref(sc)))
        for k, v in kw.items():
            if k == "stage_faces":
                sc.blocks_per_sm[7] = (sc.blocks_per_sm[7] & ~1) | (1 if v else 0)
            elif k == "stage_tables":
                sc.blocks_per_sm[7] = (sc.blocks_per_sm[7] & ~2) | (2 if v else 0)
            elif k == "blocks_per_sm":
                items = v.items() if isinstance(v, dict) else zip(STAGES, v)
                for name, b in items:
                    sc.blocks_per_sm[STAGES.index(name)] = int(b)
            else:
                setattr(sc, k, int(v))
        self._check(lib().emx_set_schedule(self.h, C.byref(sc)))

    def set_profile(self, on):
        self._check(lib().emx_set_profile(self.h, int(on)))

    def profile(self):
        """dict(ms = {stage: ms, "refill": ms, "all_step_kernels": ms}, lanes = {stage: slots processed},
        attempts = substep attempts of the field propagation, launches, iterations_launched) of the last transport"""
        ms = (C.c_double * 9)()
        nl, ni = C.c_long(), C.c_long()
        self._check(lib().emx_get_profile(self.h, C.cast(ms, C.c_void_p), C.cast(C.byref(nl), C.c_void_p),
                                          C.cast(C.byref(ni), C.c_void_p)))
        lanes = (C.c_uint64 * 8)()
        lib().emx_get_lanes(self.h, C.cast(lanes, C.c_void_p))
        return dict(ms=dict(zip(STAGES + ["refill", "all_step_kernels"], list(ms))), lanes=dict(zip(STAGES, list(lanes)[:7])),
                    attempts=int(lanes[7]), launches=nl.value, iterations_launched=ni.value)

    def iteration_times(self, max_iter=1 << 16):
        """(n, 2) float32: refill ms, step-kernel ms per iteration of the last transport (profiling on)"""
        out = np.zeros((max_iter, 2), dtype=np.float32)
        n = lib().emx_get_iteration_times(self.h, _hp(out), max_iter)
        return out[:max(n, 0)]

    def iteration_log(self, max_iter=1 << 16):
        out = np.zeros((max_iter, 2), dtype=np.uint32)
        n = lib().emx_get_iteration_log(self.h, _hp(out), max_iter)
        return out[:max(n, 0)]

    def step_batch(self, tracks, seed):
        """tracks: ctypes array of Track-compatible structs (host).  Returns a ctypes array of StepResult."""
        torch = _torch()
        n = len(tracks)
        out = (StepResult * n)()
        if n == 0:
            return out
        tin = torch.frombuffer(bytearray(bytes(tracks)), dtype=torch.uint8).cuda()
        tout = torch.empty(n * C.sizeof(StepResult), dtype=torch.uint8, device="cuda")
        self._check(lib().emx_step_batch(self.h, seed, n, C.c_void_p(tin.data_ptr()), C.c_void_p(tout.data_ptr()), _stream()))
        torch.cuda.synchronize()
        host = tout.cpu().numpy()          # keep the host copy alive while ctypes reads from it
        C.memmove(out, host.ctypes.data, n * C.sizeof(StepResult))
        del host
        return out


def field_substep_batch(problem, x, u, kappa, h):
    """Level-2 hook: one rk4_doubling substep per state in the problem's field.  Returns (x1, u1, err)."""
    torch = _torch()
    n = len(kappa)
    dev = lambda a: torch.from_numpy(_np(a, np.float64)).cuda()
    xd, ud, kd, hd = dev(x), dev(u), dev(kappa), dev(h)
    x1, u1 = torch.empty(n, 3, dtype=torch.float64, device="cuda"), torch.empty(n, 3, dtype=torch.float64, device="cuda")
    err = torch.empty(n, dtype=torch.float64, device="cuda")
    ptr = lambda t: C.c_void_p(t.data_ptr())
    problem._check(lib().emx_field_substep_batch(problem.h, n, ptr(xd), ptr(ud), ptr(kd), ptr(hd), ptr(x1), ptr(u1), ptr(err), _stream()))
    return x1.cpu().numpy(), u1.cpu().numpy(), err.cpu().numpy()


def philox_batch(ctr, key):
    torch = _torch()
    c = torch.from_numpy(_np(ctr, np.uint32).view(np.int32)).cuda()
    k = torch.from_numpy(_np(key, np.uint32).view(np.int32)).cuda()
    n = c.numel() // 4
    o = torch.empty(4 * n, dtype=torch.int32, device="cuda")
    rc = lib().emx_philox_batch(n, C.c_void_p(c.data_ptr()), C.c_void_p(k.data_ptr()), C.c_void_p(o.data_ptr()), _stream())
    if rc < 0:
        raise EmxError("emx_philox_batch %d" % rc)
    return o.cpu().numpy().view(np.uint32).reshape(n, 4)


def draw_batch(seed, prim, tid, step, nn):
    torch = _torch()
    n = len(prim)
    dev = lambda a, dt, vt: torch.from_numpy(_np(a, dt).view(vt)).cuda()
    p, t = dev(prim, np.uint32, np.int32), dev(tid, np.uint64, np.int64)
    s, q = dev(step, np.uint32, np.int32), dev(nn, np.uint32, np.int32)
    u = torch.empty(n, dtype=torch.float64, device="cuda")
    ch = torch.empty(n, dtype=torch.int64, device="cuda")
    ptr = lambda x: C.c_void_p(x.data_ptr())
    rc = lib().emx_draw_batch(seed, n, ptr(p), ptr(t), ptr(s), ptr(q), ptr(u), ptr(ch), _stream())
    if rc < 0:
        raise EmxError("emx_draw_batch %d" % rc)
    return u.cpu().numpy(), ch.cpu().numpy().view(np.uint64)


def refill_plan(alive, capacity, n_queue, static=False):
    """Level-1 hook: returns (src[capacity] int32, (new_n_live, new_n_queue, n_unfilled_holes)).
    static=True: emx_refill_plan_static, the variant that allocates nothing (capacity <= refill_plan_static_max())."""
    torch = _torch()
    a = torch.from_numpy(_np(alive, np.uint8)).cuda()
    src = torch.empty(capacity, dtype=torch.int32, device="cuda")
    counts = (C.c_long * 3)()
    name = "emx_refill_plan_static" if static else "emx_refill_plan"
    rc = getattr(lib(), name)(len(alive), capacity, n_queue, C.c_void_p(a.data_ptr()) if len(alive) else None,
                              C.c_void_p(src.data_ptr()), C.cast(counts, C.c_void_p), _stream())
    if rc < 0:
        raise EmxError("%s %d: %s" % (name, rc, (lib().emx_last_error(None) or b"").decode()))
    return src.cpu().numpy(), tuple(counts)


def refill_plan_static_max():
    return int(lib().emx_refill_plan_static_max())
