"""Pins for the oracle's RNG and track identity (R5/R6)."""
import ctypes as C

import numpy as np

from conftest import golden


def _philox(emo, ctr, key):
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    emo.lib().emo_philox4x32_10(c, k, o)
    return list(o)


def test_philox_known_answers(emo):
    for row in golden("philox4x32_10_kat.txt"):
        v = [int(x, 16) for x in row]
        assert _philox(emo, v[0:4], v[4:6]) == v[6:10]


def test_philox_is_a_bijection_of_the_counter(emo):
    # distinct counters under one key never collide (Philox is a keyed permutation)
    seen = set()
    for i in range(2000):
        seen.add(tuple(_philox(emo, [i, 0, 0, 0], [1, 2])))
    assert len(seen) == 2000


def test_uniform_open_interval_and_exact_grid(emo):
    L = emo.lib()
    assert L.emo_u01(0, 0) == 2.0 ** -53
    assert L.emo_u01(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    # 52-bit grid: (k + 1/2) 2^-52 with k = top 52 bits of (wa:wb)
    assert L.emo_u01(0x80000000, 0) == 0.5 + 2.0 ** -53
    assert L.emo_u01(0, 0xFFF) == 2.0 ** -53          # low 12 bits are discarded
    assert L.emo_u01(0, 0x1000) == 1.5 * 2.0 ** -52


def test_draw_layout_matches_block_and_words(emo):
    L = emo.lib()
    seed, prim, tid, step = 0x1234567811223344, 17, 0xAABBCCDD00112233, 5
    for n in range(7):
        o = _philox(emo, [n // 2, step, tid & 0xFFFFFFFF, tid >> 32], [seed & 0xFFFFFFFF, prim])
        h = 2 * (n % 2)
        assert L.emo_draw(seed, prim, tid, step, n) == L.emo_u01(o[h], o[h + 1])
    for o_ in range(4):
        w = _philox(emo, [0xFFFFFFFF - o_, step, tid & 0xFFFFFFFF, tid >> 32], [seed & 0xFFFFFFFF, prim])
        assert L.emo_child_tid(seed, prim, tid, step, o_) == (w[0] << 32) | w[1]


def test_draws_are_uniform(emo):
    L = emo.lib()
    x = np.array([L.emo_draw(9, p, 0, 0, n) for p in range(2000) for n in range(10)])
    assert abs(x.mean() - 0.5) < 4 * (1 / 12 / x.size) ** 0.5
    h, _ = np.histogram(x, bins=20, range=(0, 1))
    chi2 = ((h - x.size / 20) ** 2 / (x.size / 20)).sum()
    assert chi2 < 50        # 19 dof
    y = x.reshape(-1, 10)
    assert abs(np.corrcoef(y[:, 0], y[:, 1])[0, 1]) < 0.1
