"""Seeded synthetic workloads: the five problems of BASELINE.json `configs`.

This module is the ONE thing the CUDA path and the oracle share: it only describes inputs
(materials as element lists, surfaces, cells, field vector, physics switches, primary arrays).
It holds none of the method's arithmetic -- no cross sections, no sampling, no geometry tests --
and imports neither implementation.  Random inputs come from numpy's PCG64 seeded per config.

Units: MeV, cm, g/cm3, tesla.  Particle codes 0 = gamma, 1 = e-, 2 = e+.
Surface types 0/1/2 = plane x/y/z = v, 3 = cylinder about z of radius v.  Sense -1: f < 0 side.
"""
import numpy as np

PX, PY, PZ, CZ = 0, 1, 2, 3

# Z, A, mass fraction; density; mean excitation energy (ICRU-37 values; compounds by Bragg additivity)
PB = dict(name="Pb", Z=[82], A=[207.2], w=[1.0], rho=11.35, I_eV=823.0)
LAR = dict(name="lAr", Z=[18], A=[39.948], w=[1.0], rho=1.396, I_eV=188.0)
SI = dict(name="Si", Z=[14], A=[28.0855], w=[1.0], rho=2.33, I_eV=173.0)
_m = 207.2 + 183.84 + 4 * 15.999
PBWO4 = dict(name="PbWO4", Z=[82, 74, 8], A=[207.2, 183.84, 15.999],
             w=[207.2 / _m, 183.84 / _m, 4 * 15.999 / _m], rho=8.28, I_eV=542.7)
BRASS = dict(name="brass", Z=[29, 30], A=[63.546, 65.38], w=[0.7, 0.3], rho=8.53, I_eV=324.4)
PVT = dict(name="PVT", Z=[1, 6], A=[1.008, 12.011], w=[0.085, 0.915], rho=1.032, I_eV=64.7)


def physics(**kw):
    ph = dict(process_mask=63, E_min=1e-3, E_max=1e4, n_E=256, E_trk=1e-3, prod_cut_cm=0.07,
              alpha_R=0.2, rho_R=0.1, lin_loss=0.01, field_eps=1e-7, max_substeps=1000,
              vacuum_step=1e3, max_steps=10000, deposit_e_at_creation=0,
              msc=0, msc_fr=0.2, msc_smin=1e-3, fluct=0, integrator=0)
    ph.update(kw)
    return ph


def _prim(n, ptype, E, pos, dirv, vol, surf):
    return dict(ptype=np.ascontiguousarray(np.broadcast_to(np.asarray(ptype, dtype=np.int32), (n,))),
                E=np.ascontiguousarray(np.broadcast_to(np.asarray(E, dtype=np.float64), (n,))),
                pos=np.ascontiguousarray(np.broadcast_to(np.asarray(pos, dtype=np.float64), (n, 3))),
                dir=np.ascontiguousarray(np.broadcast_to(np.asarray(dirv, dtype=np.float64), (n, 3))),
                vol=np.ascontiguousarray(np.broadcast_to(np.asarray(vol, dtype=np.int32), (n,))),
                surf=np.ascontiguousarray(np.broadcast_to(np.asarray(surf, dtype=np.int32), (n,))))


def prefix(prim, n):
    """First n primaries (same indices -> same keyed histories in both implementations)."""
    return {k: np.ascontiguousarray(v[:n]) for k, v in prim.items()}


def config0(n=1000):
    """Photon-only toy: 10 MeV photons in infinite Pb, Compton + photoelectric, e- deposited at birth."""
    desc = dict(name="config0_photon_toy", seed=0, materials=[PB], surfaces=[],
                volumes=[dict(surf=[], sense=[], material=0, tally=0)], field=(0.0, 0.0, 0.0),
                physics=physics(process_mask=3, E_max=100.0, n_E=200, deposit_e_at_creation=1),
                n_slots=1024, queue_capacity=1 << 16)
    return desc, _prim(n, 0, 10.0, (0, 0, 0), (0, 0, 1), 0, -1)


def _box(surf_ids, material, tally):
    return dict(surf=list(surf_ids), sense=[1, -1, 1, -1, 1, -1], material=material, tally=tally)


def config1(n=10000):
    """Full EM shower: 1 GeV e- into a 1 m Pb cube from the centre of its -z face."""
    surfaces = [(PX, -50.0), (PX, 50.0), (PY, -50.0), (PY, 50.0), (PZ, 0.0), (PZ, 100.0)]
    desc = dict(name="config1_pb_cube", seed=1, materials=[PB], surfaces=surfaces,
                volumes=[_box(range(6), 0, 0)], field=(0.0, 0.0, 0.0), physics=physics(),
                n_slots=1 << 20, queue_capacity=1 << 24)
    return desc, _prim(n, 1, 1000.0, (0, 0, 0), (0, 0, 1), 0, 4)


def _calorimeter(field):
    surfaces = []
    for k in range(50):
        surfaces.append((PZ, 0.8 * k))
        surfaces.append((PZ, 0.8 * k + 0.23))
    surfaces.append((PZ, 40.0))                      # id 100
    surfaces += [(PZ, -10.0), (PZ, 50.0)]            # 101, 102
    surfaces += [(PX, -30.0), (PX, -20.0), (PX, 20.0), (PX, 30.0)]   # 103..106
    surfaces += [(PY, -30.0), (PY, -20.0), (PY, 20.0), (PY, 30.0)]   # 107..110
    vols = []
    for layer in range(100):                         # Pb_k -> 2k, Ar_k -> 2k+1
        vols.append(_box([104, 105, 108, 109, layer, layer + 1], layer % 2, layer))
    vols.append(_box([103, 106, 107, 110, 101, 0], -1, -1))     # 100 front vacuum
    vols.append(_box([103, 106, 107, 110, 100, 102], -1, -1))   # 101 back
    vols.append(_box([103, 104, 107, 110, 0, 100], -1, -1))     # 102 left  (x in [-30,-20])
    vols.append(_box([105, 106, 107, 110, 0, 100], -1, -1))     # 103 right
    vols.append(_box([104, 105, 107, 108, 0, 100], -1, -1))     # 104 bottom (y in [-30,-20])
    vols.append(_box([104, 105, 109, 110, 0, 100], -1, -1))     # 105 top
    return dict(materials=[PB, LAR], surfaces=surfaces, volumes=vols, field=field, physics=physics(),
                n_slots=1 << 20, queue_capacity=1 << 25)


def config2(n=10000):
    """Sampling calorimeter, 50 x (2.3 mm Pb + 5.7 mm lAr), 10 GeV e- along the layer axis, no field."""
    desc = _calorimeter((0.0, 0.0, 0.0))
    desc.update(name="config2_calorimeter", seed=2)
    return desc, _prim(n, 1, 1e4, (0, 0, -0.1), (0, 0, 1), 100, -1)


def config3(n=10000):
    """Same calorimeter in a 1 T field along y; e-/gamma alternate; beam smeared by 1 mrad (R17)."""
    desc = _calorimeter((0.0, 1.0, 0.0))
    desc.update(name="config3_calorimeter_field", seed=3)
    rng = np.random.default_rng(3)
    th = rng.normal(0.0, 1e-3, size=(n, 2))
    d = np.concatenate([th, np.ones((n, 1))], axis=1)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    pt = np.where(np.arange(n) % 2 == 0, 1, 0).astype(np.int32)
    return desc, _prim(n, pt, 1e4, (0, 0, -0.1), d, 100, -1)


def barrel_radii():
    """Cylinder radii (ascending) and mats[i] = material of the cell whose OUTER radius is radii[i] (R15, R16)."""
    radii, mats = [], []
    for k in range(10):           # Si shells, inner radii equally spaced 5..100 cm, 0.03 cm thick
        r = 5.0 + k * (95.0 / 9.0)
        radii += [r, r + 0.03]
        mats += [-1, 0]           # vacuum up to the shell, then the shell
    radii += [129.0, 152.0, 177.0]
    mats += [-1, 1, -1]           # gap, PbWO4, gap
    pitch = 118.0 / 30.0          # HCAL: 30 layers over r 177..295 keeping the 50:4 thickness ratio
    brass = 5.0 * 118.0 / 162.0
    for layer in range(30):
        r0 = 177.0 + layer * pitch
        radii += [r0 + brass, 177.0 + (layer + 1) * pitch]
        mats += [2, 3]
    radii[-1] = 295.0
    return radii, mats


def config4(n=100000):
    """Throughput stress: Si tracker shells + PbWO4 ECAL + brass/scintillator HCAL in a 4 T solenoid."""
    radii, mats = barrel_radii()
    nc = len(radii)               # 83 cylinders
    surfaces = [(CZ, r) for r in radii] + [(PZ, -150.0), (PZ, 150.0)]
    vols, tally = [], 0
    for i in range(nc):
        t = -1
        if mats[i] >= 0:
            t = tally
            tally += 1
        if i == 0:
            vols.append(dict(surf=[0, nc, nc + 1], sense=[-1, 1, -1], material=mats[0], tally=t))
        else:
            vols.append(dict(surf=[i - 1, i, nc, nc + 1], sense=[1, -1, 1, -1], material=mats[i], tally=t))
    desc = dict(name="config4_barrel_stress", seed=4, materials=[SI, PBWO4, BRASS, PVT], surfaces=surfaces,
                volumes=vols, field=(0.0, 0.0, 4.0), physics=physics(E_max=1e5),
                n_slots=1 << 20, queue_capacity=1 << 26)
    rng = np.random.default_rng(4)
    xi = rng.random(size=(n, 3))
    mu = 2.0 * xi[:, 0] - 1.0
    phi = 2.0 * np.pi * xi[:, 1]
    s = np.sqrt((1.0 - mu) * (1.0 + mu))
    d = np.stack([s * np.cos(phi), s * np.sin(phi), mu], axis=1)
    E = 1e3 * 100.0 ** xi[:, 2]
    pt = np.where(np.arange(n) % 2 == 0, 1, 0).astype(np.int32)
    return desc, _prim(n, pt, E, (0, 0, 0), d, 0, -1)


# ---- the paper's own verification problem as a sixth workload -------------
GRAPHITE = dict(name="C", Z=[6], A=[12.011], w=[1.0], rho=2.0, I_eV=78.0)
TI = dict(name="Ti", Z=[22], A=[47.867], w=[1.0], rho=4.54, I_eV=233.0)
FE = dict(name="Fe", Z=[26], A=[55.845], w=[1.0], rho=7.874, I_eV=286.0)


def config5(n=100000, n_zbins=28, half_length=700.0):
    """"An idealized coarse representation of the main components of the CMS detector, comprising six
    cylindrical shells centered about the z axis up to 375 cm ... vacuum, Si, Pb, C, Ti, and Fe"; "an isotropic
    1 GeV photon point source at the origin, composed of 100 events each with 1000 photon primaries";
    observables: cumulative energy deposition over z, steps per track by particle type.
    The paper gives neither the radii nor the length: reading = radii 30 / 125 / 175 /
    275 / 325 / 375 cm, |z| < 700 cm, no field.  The z tally is realised in the geometry: every
    shell is cut into n_zbins slabs and all cells of a slab share one tally id."""
    radii = [30.0, 125.0, 175.0, 275.0, 325.0, 375.0]
    mats = [SI, PB, GRAPHITE, TI, FE]                     # shells outside the vacuum core
    nr = len(radii)
    zs = [-half_length + k * (2.0 * half_length / n_zbins) for k in range(n_zbins + 1)]
    surfaces = [(CZ, r) for r in radii] + [(PZ, z) for z in zs]
    vols = [dict(surf=[0, nr, nr + n_zbins], sense=[-1, 1, -1], material=-1, tally=-1)]   # vacuum core
    for i in range(1, nr):
        for k in range(n_zbins):
            vols.append(dict(surf=[i - 1, i, nr + k, nr + k + 1], sense=[1, -1, 1, -1], material=i - 1, tally=k))
    desc = dict(name="config5_paper_verification", seed=5, materials=mats, surfaces=surfaces, volumes=vols,
                field=(0.0, 0.0, 0.0), physics=physics(), n_slots=1 << 20, queue_capacity=1 << 26)
    rng = np.random.default_rng(5)
    xi = rng.random(size=(n, 2))
    mu = 2.0 * xi[:, 0] - 1.0
    phi = 2.0 * np.pi * xi[:, 1]
    s = np.sqrt((1.0 - mu) * (1.0 + mu))
    d = np.stack([s * np.cos(phi), s * np.sin(phi), mu], axis=1)
    return desc, _prim(n, 0, 1000.0, (0, 0, 0), d, 0, -1)


def config6(n=20000):
    """SURVEY 8(f) f4, "non-uniform field maps" ("arbitrary magnetic fields"): the barrel of config
    4 in a solenoid field that falls off towards the ends of the barrel, B_z(0, z) = 4 T / (1 + exp((|z| - 100
    cm) / 15 cm)), with the radial component that keeps div B = 0 to first order in r (include/emx.h:
    emx_set_field_fringe).  Same primaries as config 4."""
    desc, prim = config4(n)
    desc.update(name="config6_barrel_fringe_field", seed=6, field_fringe=(100.0, 15.0))
    return desc, prim


def config7(n=10000):
    """SURVEY 8(f) f2, multiple scattering of e+- (Urban / WentzelVI "in progress") and energy-loss
    fluctuations: the sampling calorimeter and beam of config 2 with the multiple-scattering step limit and
    deflection of DESIGN.md R-MSC (f_r = 0.2, s_min = 10 um) and the fluctuations of R-FLUCT switched on."""
    desc, prim = config2(n)
    desc.update(name="config7_calorimeter_msc", seed=7,
                physics=physics(msc=1, msc_fr=0.2, msc_smin=1e-3, fluct=1))
    return desc, prim


CONFIGS = [config0, config1, config2, config3, config4, config5, config6, config7]


def get(k, n=None):
    return CONFIGS[k]() if n is None else CONFIGS[k](n)
