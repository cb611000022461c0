"""Pins of the oracle's Philox4x32-10 and uniform mapping."""
import os

import numpy as np

from paper_2209_15445_b200.inputs import philox as np_philox

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _kat():
    rows = []
    for line in open(os.path.join(GOLD, "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


def test_known_answers(ob):
    for ctr, key, want in _kat():
        c = np.array(ctr, dtype=np.uint32)
        k = np.array(key, dtype=np.uint32)
        out = np.zeros(4, dtype=np.uint32)
        ob.lib.orc_philox(c.ctypes.data, k.ctypes.data, out.ctypes.data)
        assert [int(x) for x in out] == want


def test_uniform_golden(ob):
    for line in open(os.path.join(GOLD, "closed_form_pins.txt")):
        p = line.split()
        if p and p[0] == "uniform":
            assert ob.lib.orc_uniform(1, 0, 0, 0, int(p[1])) == float(p[2])


def test_against_independent_numpy_implementation(ob):
    rng = np.random.default_rng(5)
    for _ in range(50):
        ev, seed, step = (int(x) for x in rng.integers(0, 2 ** 32, 3))
        tid = int(rng.integers(0, 2 ** 63)) * 2 + 1
        u = np_philox.uniforms(ev, seed, tid, step, 9)
        for n in range(9):
            assert ob.lib.orc_uniform(ev, seed, tid, step, n) == u[n]


def test_uniform_open_interval_and_moments(ob):
    u = np.array([ob.lib.orc_uniform(3, 1, i, 7, n) for i in range(20000) for n in range(2)])
    assert u.min() > 0.0 and u.max() <= 1.0
    assert abs(u.mean() - 0.5) < 4 * (1 / 12 / u.size) ** 0.5
    assert abs(u.var() - 1 / 12) < 5e-3
    # consecutive draws uncorrelated
    assert abs(np.corrcoef(u[0::2], u[1::2])[0, 1]) < 0.03


def test_child_ids_distinct_and_keyed(ob):
    ids = {ob.lib.orc_child_id(1, 1, p, s, c) for p in range(50) for s in range(20) for c in range(2)}
    assert len(ids) == 50 * 20 * 2
    # child id = words 0,1 of the parent's block 0xFFFFFFFF - child (R3), checked through numpy Philox
    w = np_philox.philox4x32_10(np.array([7, 0, 3, 0xFFFFFFFF - 1], dtype=np.uint32), np.array([9, 1], dtype=np.uint32))
    assert ob.lib.orc_child_id(9, 1, 7, 3, 1) == int(w[0]) | (int(w[1]) << 32)
