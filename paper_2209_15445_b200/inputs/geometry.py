"""Flat geometry descriptions for the synthetic workloads.

A geometry is a tree of placed solids in which every logical volume is placed once, so a single
u32 *touchable id* (= index into these arrays) is the whole navigation state.
Volumes are ordered so that the daughters of a volume are contiguous and in index order.
`rot`/`trans` are the *global* (world-frame) transform of each touchable, flattened on the host
(SURVEY.md §7 "flatten transforms per touchable"): local = rot^T (global - trans).
"""
from dataclasses import dataclass
import math

import numpy as np

BOX, TUBE = 0, 1


@dataclass
class Geometry:
    solid: np.ndarray            # int32 [n]      BOX | TUBE
    dims: np.ndarray             # float64 [n,3]  box: hx,hy,hz ; tube: rmin,rmax,hz
    material: np.ndarray         # int32 [n]      index into the material list
    mother: np.ndarray           # int32 [n]      -1 for the world (volume 0)
    daughter_begin: np.ndarray   # int32 [n]
    daughter_count: np.ndarray   # int32 [n]
    rot: np.ndarray              # float64 [n,9]  row-major 3x3, columns = local axes in world frame
    trans: np.ndarray            # float64 [n,3]
    material_names: list
    name: str = ""

    @property
    def n_volumes(self):
        return int(self.solid.shape[0])


def _finish(solid, dims, material, mother, rot, trans, material_names, name):
    n = len(solid)
    mother = np.asarray(mother, dtype=np.int32)
    begin = np.zeros(n, dtype=np.int32)
    count = np.zeros(n, dtype=np.int32)
    for v in range(1, n):
        m = mother[v]
        if count[m] == 0:
            begin[m] = v
        assert begin[m] + count[m] == v, "daughters must be contiguous"
        count[m] += 1
    return Geometry(np.asarray(solid, dtype=np.int32), np.ascontiguousarray(dims, dtype=np.float64),
                    np.asarray(material, dtype=np.int32), mother, begin, count,
                    np.ascontiguousarray(rot, dtype=np.float64).reshape(n, 9),
                    np.ascontiguousarray(trans, dtype=np.float64), list(material_names), name)


def calorimeter(n_layers=50, t_abs=0.23, t_gap=0.57):
    """Configs 1-3 (BASELINE.json:configs[0..2]; PAPER.md:61 layer structure, Pb instead of PbWO4).

    Volumes: 0 world, 1 calorimeter, 2..51 layers, 52+2i absorber (Pb) of layer i, 53+2i gap (LAr).
    Materials: 0 vacuum, 1 Pb, 2 LAr.
    """
    t_layer = t_abs + t_gap
    length = n_layers * t_layer
    solid, dims, material, mother, trans = [], [], [], [], []

    def add(h, mat, mom, centre):
        solid.append(BOX); dims.append(h); material.append(mat); mother.append(mom); trans.append(centre)

    add((40.0, 30.0, 30.0), 0, -1, (20.0, 0.0, 0.0))                       # x in [-20, 60]
    add((0.5 * length, 20.0, 20.0), 0, 0, (0.5 * length, 0.0, 0.0))        # x in [0, 40]
    for i in range(n_layers):
        add((0.5 * t_layer, 20.0, 20.0), 0, 1, (t_layer * i + 0.5 * t_layer, 0.0, 0.0))
    for i in range(n_layers):
        add((0.5 * t_abs, 20.0, 20.0), 1, 2 + i, (t_layer * i + 0.5 * t_abs, 0.0, 0.0))
        add((0.5 * t_gap, 20.0, 20.0), 2, 2 + i, (t_layer * i + t_abs + 0.5 * t_gap, 0.0, 0.0))
    n = len(solid)
    rot = np.tile(np.eye(3).reshape(1, 9), (n, 1))
    return _finish(solid, dims, material, mother, rot, trans, ["vacuum", "Pb", "LAr"], "calorimeter")


def barrel(n_eta=170, n_phi=360, n_shells=10, crystal="PbWO4"):
    """Configs 4-5 (BASELINE.json:configs[3]; SURVEY.md §8(d) cfg 4).

    Volumes: 0 world tube, 1..10 Si shells, 11 ECAL mother tube, 12 + i*n_phi + j crystal (row i, col j).
    Materials: 0 vacuum, 1 Si, 2 `crystal`: "PbWO4" (the effective element Z=73 of BASELINE.json:configs[3]) or
    "PbWO4_true" (the compound Pb + W + 4 O).
    """
    solid, dims, material, mother, trans, rot = [], [], [], [], [], []
    eye = np.eye(3)

    def add(kind, d, mat, mom, t, r):
        solid.append(kind); dims.append(d); material.append(mat); mother.append(mom)
        trans.append(t); rot.append(np.asarray(r).reshape(9))

    add(TUBE, (0.0, 300.0, 300.0), 0, -1, (0, 0, 0), eye)
    for s in range(n_shells):
        r_in = 3.0 + 107.0 * s / 9.0
        add(TUBE, (r_in, r_in + 0.03, 280.0), 1, 0, (0, 0, 0), eye)
    add(TUBE, (127.5, 153.0, 290.0), 0, 0, (0, 0, 0), eye)
    mom = 1 + n_shells
    delta = 2.0 * math.pi / 360.0
    for i in range(n_eta):
        eta = (i - 0.5 * (n_eta - 1)) * delta
        theta = 2.0 * math.atan(math.exp(-eta))
        st, ct = math.sin(theta), math.cos(theta)
        for j in range(n_phi):
            phi = (j + 0.5) * delta
            sp, cp = math.sin(phi), math.cos(phi)
            a = np.array([st * cp, st * sp, ct])
            xh = np.array([-sp, cp, 0.0])
            yh = np.cross(a, xh)
            front = np.array([129.0 * cp, 129.0 * sp, 129.0 * ct / st])
            R = np.stack([xh, yh, a], axis=1)            # columns = local axes
            add(BOX, (1.1, 1.1, 11.5), 2, mom, front + 11.5 * a, R)
    return _finish(solid, dims, material, mother, np.stack(rot), trans,
                   ["vacuum", "Si", crystal], "barrel")
