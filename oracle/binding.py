"""ORACLE -- TEST INFRASTRUCTURE ONLY.  ctypes binding of oracle/liboracle.so (oracle/oracle.h)."""
import ctypes as C

import numpy as np

from . import build as _build

TRACK = np.dtype([("pos", "f8", 3), ("dir", "f8", 3), ("ekin", "f8"), ("id", "u8"), ("event", "u4"),
                  ("step", "u4"), ("volume", "u4"), ("species", "i4")], align=True)
RESULT = np.dtype([("post", TRACK), ("alive", "i4"), ("outcome", "i4"), ("n_sec", "i4"), ("chords", "i4"),
                   ("s", "f8"), ("edep_dep", "f8"), ("edep_cut", "f8"), ("escaped", "f8"), ("killed", "f8")],
                  align=True)
assert TRACK.itemsize == 80 and RESULT.itemsize == 136

OUTCOMES = ["boundary", "compton", "pair", "photo", "brem", "ioni", "anni", "stopped", "truncated", "loss",
            "escaped", "killed", "closed"]

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class Geometry(C.Structure):
    _fields_ = [("n_vol", C.c_int32), ("solid", _ip), ("dims", _dp), ("material", _ip), ("mother", _ip),
                ("daughter_begin", _ip), ("daughter_count", _ip), ("rot", _dp), ("trans", _dp)]


class Materials(C.Structure):
    _fields_ = [("n_mat", C.c_int32), ("tables", _dp), ("scalars", _dp), ("n_elem", _ip), ("elem_bk", _dp), ("pe_cum", _dp)]


class Field(C.Structure):
    _fields_ = [("kind", C.c_int32), ("B", C.c_double * 3), ("nr", C.c_int32), ("nz", C.c_int32),
                ("r0", C.c_double), ("z0", C.c_double), ("dr", C.c_double), ("dz", C.c_double), ("bz", _dp)]


class Config(C.Structure):
    _fields_ = [("delta_chord", C.c_double), ("eps_push", C.c_double), ("alpha_R", C.c_double),
                ("rho_R", C.c_double), ("chord_budget", C.c_int32), ("seed", C.c_uint32),
                ("max_steps", C.c_uint32), ("reserved", C.c_int32)]


class Ledger(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("deposited", "below_cut", "escaped", "killed", "primary")]

    def total(self):
        return self.deposited + self.below_cut + self.escaped + self.killed


class Stats(C.Structure):
    _fields_ = [("steps", C.c_uint64 * 3), ("outcomes", C.c_uint64 * 13), ("secondaries", C.c_uint64 * 3),
                ("chords", C.c_uint64), ("peak_stack", C.c_uint64), ("iterations", C.c_uint64)]


def _lib():
    lib = C.CDLL(_build.build())
    vp = C.c_void_p
    d, i32, u32, u64 = C.c_double, C.c_int32, C.c_uint32, C.c_uint64
    sig = {
        "orc_create": (vp, [C.POINTER(Geometry), C.POINTER(Materials), C.POINTER(Field), C.POINTER(Config)]),
        "orc_destroy": (None, [vp]),
        "orc_philox": (None, [vp, vp, vp]),
        "orc_uniform": (d, [u32, u32, u64, u32, u32]),
        "orc_child_id": (u64, [u32, u32, u64, u32, u32]),
        "orc_lookup": (d, [vp, i32, i32, d]),
        "orc_inverse_range": (d, [vp, i32, i32, d]),
        "orc_distance": (d, [vp, vp, vp, u32, d]),
        "orc_locate": (C.c_int64, [vp, vp]),
        "orc_inside": (i32, [vp, vp, u32]),
        "orc_solid_entry": (d, [i32, vp, vp, vp]),
        "orc_solid_exit": (d, [i32, vp, vp, vp]),
        "orc_propagate": (i32, [vp, i32, d, vp, vp, u32, d, vp, vp, vp]),
        "orc_helix": (None, [vp, i32, d, d, vp, vp, vp, vp]),
        "orc_rk4": (None, [vp, i32, d, d, vp, vp, vp, vp]),
        "orc_field_at": (None, [vp, vp, vp]),
        "orc_rotate": (None, [vp, d, d, d, vp]),
        "orc_interact": (None, [vp, i32, vp, i32, vp, vp]),
        "orc_step": (None, [vp, vp, vp, vp]),
        "orc_place": (C.c_int64, [vp, vp, vp]),
        "orc_run": (i32, [vp, C.c_size_t, vp, vp, C.POINTER(Ledger), C.POINTER(Stats)]),
        "orc_set_recorder": (None, [vp, u32, u32, vp, C.c_size_t]),
        "orc_recorded": (C.c_size_t, [vp]),
        "orc_build_material": (None, [d, d, d, vp, vp]),
        "orc_build_compound": (None, [i32, vp, vp, vp, d, vp, vp, vp, vp]),
        "orc_sigma_compton": (d, [d]), "orc_pair_shape": (d, [d]), "orc_sigma_photo": (d, [d, d]),
        "orc_brem_shape": (d, [d, d]), "orc_srad_shape": (d, [d, d]), "orc_sigma_moller": (d, [d, d]),
        "orc_sigma_bhabha": (d, [d, d]), "orc_sigma_annihilation": (d, [d]),
        "orc_s_coll": (d, [d, d, d, d, d, i32]),
    }
    for name, (res, args) in sig.items():
        f = getattr(lib, name)
        f.restype, f.argtypes = res, args
    return lib


lib = _lib()


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _v3(x):
    return np.ascontiguousarray(x, dtype=np.float64).reshape(3)


class Oracle:
    """One oracle context: geometry + materials + field + config, copied at construction."""

    def __init__(self, geom, tables, scalars, field, delta_chord=1e-3, eps_push=1e-7, alpha_R=0.2, rho_R=0.1,
                 chord_budget=16, seed=1, max_steps=1000000, elements=None):
        """elements: None (single-element materials) or (n_elem[n_mat], elem_bk[n_mat,4], pe_cum[n_mat,2048,4])."""
        g = Geometry(geom.n_volumes, geom.solid.ctypes.data_as(_ip), geom.dims.ctypes.data_as(_dp),
                     geom.material.ctypes.data_as(_ip), geom.mother.ctypes.data_as(_ip),
                     geom.daughter_begin.ctypes.data_as(_ip), geom.daughter_count.ctypes.data_as(_ip),
                     geom.rot.ctypes.data_as(_dp), geom.trans.ctypes.data_as(_dp))
        tables = np.ascontiguousarray(tables, dtype=np.float64)
        scalars = np.ascontiguousarray(scalars, dtype=np.float64)
        if elements is None:
            m = Materials(tables.shape[0], tables.ctypes.data_as(_dp), scalars.ctypes.data_as(_dp), None, None, None)
        else:
            ne = np.ascontiguousarray(elements[0], dtype=np.int32)
            bk = np.ascontiguousarray(elements[1], dtype=np.float64)
            cum = np.ascontiguousarray(elements[2], dtype=np.float64)
            assert ne.shape == (tables.shape[0],) and bk.shape == (tables.shape[0], 4) and cum.shape == (tables.shape[0], 2048, 4)
            m = Materials(tables.shape[0], tables.ctypes.data_as(_dp), scalars.ctypes.data_as(_dp), ne.ctypes.data_as(_ip),
                          bk.ctypes.data_as(_dp), cum.ctypes.data_as(_dp))
        bz = np.ascontiguousarray(field.bz, dtype=np.float64)
        f = Field(field.kind, (C.c_double * 3)(*field.B), field.nr, field.nz, field.r0, field.z0, field.dr,
                  field.dz, bz.ctypes.data_as(_dp))
        cfg = Config(delta_chord, eps_push, alpha_R, rho_R, chord_budget, seed, max_steps, 0)
        self.n_vol = geom.n_volumes
        self.seed = seed
        self.ctx = lib.orc_create(C.byref(g), C.byref(m), C.byref(f), C.byref(cfg))
        self._rec = None

    def __del__(self):
        if getattr(self, "ctx", None):
            lib.orc_destroy(self.ctx)
            self.ctx = None

    # -- primitives
    def lookup(self, mat, tab, ekin):
        return lib.orc_lookup(self.ctx, mat, tab, ekin)

    def inverse_range(self, mat, tab, r):
        return lib.orc_inverse_range(self.ctx, mat, tab, r)

    def distance(self, pos, direc, volume, s_max=np.inf):
        return lib.orc_distance(self.ctx, _p(_v3(pos)), _p(_v3(direc)), volume, s_max)

    def locate(self, pos):
        return lib.orc_locate(self.ctx, _p(_v3(pos)))

    def inside(self, pos, volume):
        return bool(lib.orc_inside(self.ctx, _p(_v3(pos)), volume))

    def field_at(self, pos):
        b = np.zeros(3)
        lib.orc_field_at(self.ctx, _p(_v3(pos)), _p(b))
        return b

    def rk4(self, charge, pmom, h, pos, direc):
        p1, d1 = np.zeros(3), np.zeros(3)
        lib.orc_rk4(self.ctx, charge, pmom, h, _p(_v3(pos)), _p(_v3(direc)), _p(p1), _p(d1))
        return p1, d1

    def propagate(self, charge, ekin, pos, direc, volume, s_phys):
        p, d, push = _v3(pos).copy(), _v3(direc).copy(), np.zeros(3)
        s, ch = C.c_double(0), C.c_int32(0)
        flag = lib.orc_propagate(self.ctx, charge, ekin, _p(p), _p(d), volume, s_phys, C.byref(s), C.byref(ch), _p(push))
        return flag, p, d, s.value, ch.value, push

    # -- tracks
    def make_tracks(self, prim):
        """Primaries dict (inputs.primaries) -> TRACK array; id = index within the event; placed by G5."""
        n = len(prim["ekin"])
        t = np.zeros(n, dtype=TRACK)
        t["pos"], t["dir"], t["ekin"] = prim["pos"], prim["dir"], prim["ekin"]
        t["event"], t["species"] = prim["event"], prim["species"]
        ev = prim["event"]
        first = np.r_[True, ev[1:] != ev[:-1]]
        start = np.maximum.accumulate(np.where(first, np.arange(n), 0))
        t["id"] = np.arange(n) - start
        for i in range(n):
            v = lib.orc_place(self.ctx, _p(t["pos"][i].copy()), _p(t["dir"][i].copy()))
            assert v >= 0, "primary outside the world"
            t["volume"][i] = v
        return t

    def step(self, tracks):
        """One step per track -> (RESULT array, secondaries TRACK array [n,2])."""
        tracks = np.ascontiguousarray(tracks, dtype=TRACK)
        n = tracks.shape[0]
        res = np.zeros(n, dtype=RESULT)
        sec = np.zeros((n, 2), dtype=TRACK)
        base_t, base_r, base_s = tracks.ctypes.data, res.ctypes.data, sec.ctypes.data
        for i in range(n):
            lib.orc_step(self.ctx, base_t + 80 * i, base_r + 136 * i, base_s + 160 * i)
        return res, sec

    def interact(self, process, tracks, material):
        tracks = np.ascontiguousarray(tracks, dtype=TRACK)
        n = tracks.shape[0]
        res = np.zeros(n, dtype=RESULT)
        sec = np.zeros((n, 2), dtype=TRACK)
        for i in range(n):
            lib.orc_interact(self.ctx, process, tracks.ctypes.data + 80 * i, material, res.ctypes.data + 136 * i,
                             sec.ctypes.data + 160 * i)
        return res, sec

    def set_recorder(self, mask, stride, cap):
        self._rec = np.zeros(cap, dtype=TRACK)
        lib.orc_set_recorder(self.ctx, mask, stride, _p(self._rec), cap)

    def recorded(self):
        return self._rec[:lib.orc_recorded(self.ctx)].copy()

    def run(self, tracks, edep=None):
        """Full transport -> (edep[n_vol], Ledger, Stats)."""
        tracks = np.ascontiguousarray(tracks, dtype=TRACK)
        if edep is None:
            edep = np.zeros(self.n_vol)
        led, st = Ledger(), Stats()
        lib.orc_run(self.ctx, tracks.shape[0], _p(tracks), _p(edep), C.byref(led), C.byref(st))
        return edep, led, st


def build_material(Z, A, rho):
    tab = np.zeros((12, 2048))
    scal = np.zeros(8)
    lib.orc_build_material(Z, A, rho, _p(tab), _p(scal))
    return tab, scal


def build_compound(Z, A, nu, rho):
    """-> (tables[12,2048], scalars[8], elem_bk[4], pe_cum[2048,4]) of a compound with nu[i] atoms of (Z[i], A[i])."""
    Z, A, nu = (np.ascontiguousarray(x, dtype=np.float64) for x in (Z, A, nu))
    tab, scal, bk, cum = np.zeros((12, 2048)), np.zeros(8), np.zeros(4), np.zeros((2048, 4))
    lib.orc_build_compound(len(Z), _p(Z), _p(A), _p(nu), rho, _p(tab), _p(scal), _p(bk), _p(cum))
    return tab, scal, bk, cum
