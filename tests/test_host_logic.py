"""Host-side logic that needs no GPU: the ray-cast camera and picture writer, bench.py's workload naming and
event sharding, and the binding's description of the C structures."""
import argparse
import importlib.util
import os

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_raycast_cameras_and_ppm(tmp_path):
    from paper_2209_15445_b200 import raycast
    p, d = raycast.barrel_rays(16, 8)
    assert p.shape == d.shape == (128, 3) and not p.any()
    np.testing.assert_allclose(np.linalg.norm(d, axis=1), 1.0, rtol=0, atol=1e-15)
    eta = -np.log(np.tan(0.5 * np.arccos(d[:, 2])))
    assert abs(eta).max() < 1.45 and np.allclose(eta.reshape(8, 16)[:, 0], eta.reshape(8, 16)[:, 5])   # rows = eta
    phi = np.arctan2(d[:, 1], d[:, 0]) % (2 * np.pi)
    assert np.allclose(np.diff(phi.reshape(8, 16)[0]), 2 * np.pi / 16)                                   # columns = phi
    p, d = raycast.calorimeter_rays(4, 2)
    assert (p[:, 0] == -10.0).all() and (d == [1.0, 0.0, 0.0]).all() and abs(p[:, 1:]).max() < 25.0
    out = tmp_path / "x.ppm"
    raycast.write_ppm(str(out), np.arange(8.0), 4, 2)
    data = out.read_bytes()
    head = b"P6\n4 2\n255\n"
    assert data.startswith(head) and len(data) == len(head) + 24
    assert data[len(head):len(head) + 3] == b"\x00\x00\x00" and data[-3:] == b"\xff\xff\xff"


def test_bench_workloads_and_sharding():
    b = _bench()
    a = argparse.Namespace(config=2, events=10000, field=0.0, max_steps=1000000)
    assert b.workload_name(a).startswith("config2: 10000 x 10 GeV e-")
    a = argparse.Namespace(config=3, events=10000, field=1.0, max_steps=1000000)
    assert "uniform 1.0 T" in b.workload_name(a)
    a = argparse.Namespace(config=4, events=100, field=0.0, max_steps=4096)
    assert "max_steps=4096" in b.workload_name(a) and "61200" in b.workload_name(a)
    a = argparse.Namespace(config=3, events=10000, field=1.0, max_steps=1000000, species="gamma")
    assert "10 GeV gamma" in b.workload_name(a)
    a = argparse.Namespace(config=1, events=256, field=0.0, max_steps=1000000, species="e-", e_primary=1000.0, spread=0.0)
    assert b.workload_name(a).startswith("config1: 256 x 1 GeV e-")
    _, _, _, _, p1 = b.workload(a)
    assert len(p1["ekin"]) == 256 and (p1["ekin"] == 1000.0).all() and not p1["pos"].any()
    # ranks own disjoint, consecutive event ranges: Philox streams are keyed by event id
    assert [b.shard_first_event(r, 10000) for r in range(4)] == [0, 10000, 20000, 30000]
    assert b.BYTES_PER_STEP == 76 + 76 + 8
    t = b.ncu_traffic()
    assert t is None or (set(b.KERNELS) <= set(t["kernels"]) <= set(b.KERNELS) | {"move_kernel"} and t.get("commit"))
    if t is not None:      # the merged move kernel: its own row, or the sum of its two bodies
        m = b.traffic_of(t, "move_kernel")
        # captures of launches at the peak of a pass (the file names the population step of each): within 1 % of each other
        bodies = t["kernels"]["gamma_move_kernel"]["tracks"] + t["kernels"]["charged_move_kernel"]["tracks"]
        assert abs(m["tracks"] - bodies) <= 0.01 * bodies
        assert m["dram_bytes"] == m["dram_read"] + m["dram_write"] > t["kernels"]["gamma_move_kernel"]["dram_bytes"]
    g, tabs, scal, fld, prim = b.workload(argparse.Namespace(config=2, events=7, field=0.0), first_event=3)
    assert list(prim["event"]) == list(range(3, 10)) and (prim["ekin"] == 10000.0).all() and g.n_volumes == 152


def test_interaction_outcomes_match_the_header():
    from paper_2209_15445_b200 import adept
    names = {}
    for line in open(os.path.join(ROOT, "include", "adept.h")):
        for part in line.split(","):
            part = part.strip()
            if part.startswith("ADEPT_OUT_") and "=" in part:
                k, v = part.split("=")
                names[k.strip()] = int(v.strip().split()[0])
    want = {names[k] for k in ("ADEPT_OUT_COMPTON", "ADEPT_OUT_PAIR", "ADEPT_OUT_BREM", "ADEPT_OUT_IONI", "ADEPT_OUT_ANNI",
                               "ADEPT_OUT_CLOSED")}
    assert set(adept.INTERACTION_OUTCOMES) == want
