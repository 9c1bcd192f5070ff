"""Host logic of the CUDA library without a device: the candidate lists that `neighbour()` walks after a boundary
crossing (C8; include/emx.h emx_neighbour_candidates) are pruned of the cells a parallel face of their own
keeps on the other side of the surface crossed.  Pruning must never remove the cell the definition names -- the
ORACLE's full scan in id order over all cells -- for points on the surface or within the landing tolerance of it."""
import numpy as np
import pytest

from paper_2203_09467_b200 import workloads as W
from states import bounding_box


def _points_on(stype, v, lo, hi, rng, n):
    x = rng.uniform(lo, hi, size=(n, 3))
    if stype < 3:
        x[:, stype] = v
    else:
        phi = rng.uniform(0, 2 * np.pi, n)
        x[:, 0], x[:, 1] = v * np.cos(phi), v * np.sin(phi)
    return x


def _normal(stype, x):
    g = np.zeros(3)
    if stype < 3:
        g[stype] = 1.0
    else:
        g[:2] = x[:2] / np.hypot(x[0], x[1])
    return g


@pytest.mark.parametrize("cfg", [1, 2, 4, 5])
def test_pruned_candidate_lists_keep_the_cell_of_the_full_scan(emo, cfg):
    from paper_2203_09467_b200 import emx
    desc, _ = W.get(cfg, 4)
    G = emx.Problem(desc, build=False)            # host description only: no device needed
    O = emo.Problem(desc)
    lo, hi = bounding_box(desc)
    rng = np.random.default_rng(100 + cfg)
    eps = desc["physics"]["field_eps"]
    n_vol = len(desc["volumes"])
    surfaces = list(enumerate(desc["surfaces"]))
    if len(surfaces) > 24:                        # a spread of inner and outer surfaces
        pick = sorted(set(rng.choice(len(surfaces), 16, replace=False).tolist()) | set(range(len(surfaces) - 8, len(surfaces))))
        surfaces = [surfaces[k] for k in pick]
    found = escaped = 0
    for S, (stype, v) in surfaces:
        cand = {s: np.concatenate([G.neighbour_candidates(S, s, 0), G.neighbour_candidates(S, s, 1)]) for s in (1, -1)}
        listing = {s: set(G.neighbour_candidates(S, s, 0).tolist()) for s in (1, -1)}
        for s in (1, -1):                         # the first list really is "cells that list (S, s)"
            for c in listing[s]:
                vol = desc["volumes"][c]
                assert (S, s) in zip(vol["surf"], vol["sense"])
            assert len(cand[s]) == len(set(cand[s].tolist())) <= n_vol
        for x in _points_on(stype, v, lo, hi, rng, 60):
            nrm = _normal(stype, x)
            u = rng.normal(size=3)
            u /= np.linalg.norm(u)
            if abs(u @ nrm) < 1e-3:
                continue
            s = 1 if u @ nrm > 0 else -1
            for off in (0.0, eps, -eps):          # on the surface, and a landing tolerance short of / beyond it
                xx = x + off * nrm
                nv = O.neighbour(xx, u, S)
                if nv >= 0:
                    assert nv in cand[s], (cfg, S, s, off, nv)
                    found += 1
                else:
                    escaped += 1
    assert found > 100 and escaped > 0
    # the point of the pruning: leaving the world through an outer surface there is nothing to test
    if cfg in (2, 4):
        outer = {2: (102, 1), 4: (82, 1)}[cfg]    # z = 50 cm plane of the calorimeter world; outermost cylinder
        assert len(G.neighbour_candidates(outer[0], outer[1], 0)) == 0
        assert len(G.neighbour_candidates(outer[0], outer[1], 1)) == 0


def test_argument_checks():
    from paper_2203_09467_b200 import emx
    desc, _ = W.get(1, 4)
    G = emx.Problem(desc, build=False)
    L = emx.lib()
    assert L.emx_neighbour_candidates(G.h, 99, 1, 0, None, 0) == -1
    assert L.emx_neighbour_candidates(G.h, 0, 0, 0, None, 0) == -1
    assert L.emx_neighbour_candidates(G.h, 0, 1, 2, None, 0) == -1
    assert L.emx_neighbour_candidates(G.h, 0, 1, 0, None, 4) == -1
