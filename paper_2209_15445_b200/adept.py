"""Thin ctypes binding of libadept_b200.so (include/adept.h): argument marshalling only.

Every step of the transport path runs inside the CUDA library; PyTorch supplies the device
workspace and the streams (BASELINE.json:north_star).  There is no CPU fallback: importing this
module fails loudly when the library is missing or cannot be loaded.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("ADEPT_B200_LIB", os.path.join(HERE, "libadept_b200.so"))

OK, EINVAL, ENOMEM, EOVERFLOW, ECUDA, ESTATE = 0, -1, -2, -3, -4, -5
NAV_LOOP, NAV_BVH, NAV_LOOP_F32, NAV_BVH_F32 = 0, 1, 2, 3
STATIC_MAX_RAYS = 65536  # ADEPT_STATIC_MAX_RAYS: most rays of one raycast_static call
OUTCOMES = ["boundary", "compton", "pair", "photo", "brem", "ioni", "anni", "stopped", "truncated", "loss",
            "escaped", "killed", "closed"]

TRACK = np.dtype([("pos", "f8", 3), ("dir", "f8", 3), ("ekin", "f8"), ("id", "u8"), ("event", "u4"),
                  ("step", "u4"), ("volume", "u4"), ("species", "i4")], align=True)
RESULT = np.dtype([("post", TRACK), ("alive", "i4"), ("outcome", "i4"), ("n_sec", "i4"), ("chords", "i4"),
                   ("s", "f8"), ("edep_dep", "f8"), ("edep_cut", "f8"), ("escaped", "f8"), ("killed", "f8")],
                  align=True)

_dp, _ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)


class CGeometry(C.Structure):
    _fields_ = [("n_volumes", C.c_int32), ("solid", _ip), ("dims", _dp), ("material", _ip), ("mother", _ip),
                ("daughter_begin", _ip), ("daughter_count", _ip), ("rot", _dp), ("trans", _dp)]


class CTables(C.Structure):
    _fields_ = [("data", _dp), ("n_elem", _ip), ("elem_bk", _dp), ("pe_cum", _dp)]


class CField(C.Structure):
    _fields_ = [("kind", C.c_int32), ("B", C.c_double * 3), ("nr", C.c_int32), ("nz", C.c_int32),
                ("r0", C.c_double), ("z0", C.c_double), ("dr", C.c_double), ("dz", C.c_double), ("bz", _dp)]


class CConfig(C.Structure):
    _fields_ = [("delta_chord", C.c_double), ("eps_push", C.c_double), ("alpha_R", C.c_double), ("rho_R", C.c_double),
                ("chord_budget", C.c_int32), ("seed", C.c_uint32), ("max_steps", C.c_uint32), ("navigator", C.c_int32),
                ("n_event_slots", C.c_int32), ("sync_interval", C.c_int32), ("track_capacity", C.c_uint64),
                ("leak_capacity", C.c_uint64), ("stage_capacity", C.c_uint64), ("time_kernels", C.c_int32),
                ("inject_chunk", C.c_uint64), ("pending_capacity", C.c_uint64), ("concurrent_species", C.c_int32), ("steps_per_launch", C.c_int32),
                ("use_graphs", C.c_int32), ("low_occupancy_below", C.c_int32)]


class CLedger(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("deposited", "below_cut", "escaped", "killed", "primary")]

    def total(self):
        return self.deposited + self.below_cut + self.escaped + self.killed


class CStats(C.Structure):
    _fields_ = [("steps", C.c_uint64 * 3), ("outcomes", C.c_uint64 * 13), ("secondaries", C.c_uint64 * 3),
                ("chords", C.c_uint64), ("iterations", C.c_uint64), ("peak_population", C.c_uint64),
                ("launches", C.c_uint64)]


# outcomes (ADEPT_OUT_*) counted by the interaction kernel: Compton, pair, brems, ionisation, annihilation, closed
INTERACTION_OUTCOMES = (1, 2, 4, 5, 6, 12)

EXPORTS = ["adept_last_error", "adept_default_config", "adept_workspace_bytes", "adept_init",
           "adept_enqueue_primaries", "adept_enqueue_batch", "adept_transport", "adept_transport_many",
           "adept_read_scoring", "adept_read_leaked", "adept_get_stats", "adept_get_kernel_times", "adept_set_kernel_timing", "adept_get_iteration_trace",
           "adept_raycast_batch", "adept_raycast_batch_static", "adept_buffer_create", "adept_buffer_add", "adept_buffer_flush", "adept_buffer_pending", "adept_buffer_take",
           "adept_buffer_destroy", "adept_step_frozen", "adept_step_population", "adept_reset_slot",
           "adept_distance_batch", "adept_locate_batch", "adept_relocate_batch", "adept_shutdown"]


def load_library():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2209_15445_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i, sz = C.c_void_p, C.c_int, C.c_size_t
    lib.adept_last_error.restype = C.c_char_p
    lib.adept_default_config.argtypes = [C.POINTER(CConfig)]
    lib.adept_workspace_bytes.restype = sz
    lib.adept_workspace_bytes.argtypes = [C.POINTER(CConfig), C.POINTER(CGeometry), i, C.POINTER(CField)]
    lib.adept_init.argtypes = [C.POINTER(vp), C.POINTER(CGeometry), vp, i, C.POINTER(CTables), C.POINTER(CField),
                               C.POINTER(CConfig), vp, sz]
    lib.adept_enqueue_primaries.argtypes = [vp, i, C.c_uint32, i, vp, vp, vp, vp]
    lib.adept_enqueue_batch.argtypes = [vp, i, i, vp, vp, vp, vp, vp, vp]
    lib.adept_transport.argtypes = [vp, i, vp]
    lib.adept_transport_many.argtypes = [vp, i, vp, vp]
    lib.adept_read_scoring.argtypes = [vp, i, vp, sz, C.POINTER(CLedger), vp]
    lib.adept_read_leaked.argtypes = [vp, i, vp, sz, C.POINTER(sz)]
    lib.adept_get_stats.argtypes = [vp, i, C.POINTER(CStats)]
    lib.adept_get_kernel_times.argtypes = [vp, i, vp, vp]
    lib.adept_set_kernel_timing.argtypes = [vp, i]
    lib.adept_get_iteration_trace.argtypes = [vp, i, vp, vp, sz, C.POINTER(sz)]
    lib.adept_step_frozen.argtypes = [vp, i, vp, vp, vp, vp]
    lib.adept_step_population.argtypes = [vp, i, i, vp, vp, sz, C.POINTER(sz), vp]
    lib.adept_reset_slot.argtypes = [vp, i]
    lib.adept_distance_batch.argtypes = [vp, i, i, vp, vp, vp, vp, vp, vp]
    lib.adept_locate_batch.argtypes = [vp, i, i, vp, vp, vp]
    lib.adept_relocate_batch.argtypes = [vp, i, i, vp, vp, vp, vp, vp]
    lib.adept_shutdown.argtypes = [vp]
    lib.adept_raycast_batch.argtypes = [vp, i, i, vp, vp, i, vp, vp, C.POINTER(C.c_double), vp]
    lib.adept_raycast_batch_static.argtypes = [vp, i, i, vp, vp, i, vp, vp, vp]
    lib.adept_buffer_create.argtypes = [C.POINTER(vp), vp, i, sz, vp]
    lib.adept_buffer_add.argtypes = [vp, C.c_uint32, C.c_uint64, i, vp, vp, C.c_double]
    lib.adept_buffer_flush.argtypes = [vp]
    lib.adept_buffer_pending.argtypes = [vp, C.POINTER(sz), C.POINTER(sz), C.POINTER(C.c_uint64)]
    lib.adept_buffer_take.argtypes = [vp, vp, sz, C.POINTER(CLedger), vp, sz, C.POINTER(sz)]
    lib.adept_buffer_destroy.argtypes = [vp]
    return lib


lib = load_library()


class AdeptError(RuntimeError):
    def __init__(self, code):
        self.code = code
        super().__init__(f"adept error {code}: {lib.adept_last_error().decode()}")


def _check(code):
    if code != OK:
        raise AdeptError(code)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def default_config(**over):
    cfg = CConfig()
    lib.adept_default_config(C.byref(cfg))
    for k, v in over.items():
        if not hasattr(cfg, k):
            raise TypeError(f"unknown config field {k}")
        setattr(cfg, k, v)
    return cfg


def _stream_ptr(stream):
    if stream is None:
        return None
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


class Adept:
    """One library context.  `geom`, `field` come from paper_2209_15445_b200.inputs; `scalars` is
    (n_mat, 8) and `tables` (n_mat, 12, 2048) as built by inputs.materials.build_material_set."""

    def __init__(self, geom, tables, scalars, field, device="cuda:0", _workspace_bytes=None, elements=None, **config):
        """elements: None, or (n_elem, elem_bk, pe_cum) from inputs.materials.element_tables for compound materials.
        _workspace_bytes (tests): size of the workspace handed to adept_init instead of adept_workspace_bytes()."""
        import torch
        self._torch = torch
        self.device = torch.device(device)
        self.ctx = None
        self.cfg = default_config(**config)
        self.n_volumes = geom.n_volumes
        self._keep = [geom, np.ascontiguousarray(tables, dtype=np.float64),
                      np.ascontiguousarray(scalars, dtype=np.float64),
                      np.ascontiguousarray(field.bz, dtype=np.float64)]
        g = CGeometry(geom.n_volumes, geom.solid.ctypes.data_as(_ip), geom.dims.ctypes.data_as(_dp),
                      geom.material.ctypes.data_as(_ip), geom.mother.ctypes.data_as(_ip),
                      geom.daughter_begin.ctypes.data_as(_ip), geom.daughter_count.ctypes.data_as(_ip),
                      geom.rot.ctypes.data_as(_dp), geom.trans.ctypes.data_as(_dp))
        if elements is None:
            t = CTables(self._keep[1].ctypes.data_as(_dp), None, None, None)
        else:
            el = [np.ascontiguousarray(elements[0], dtype=np.int32), np.ascontiguousarray(elements[1], dtype=np.float64),
                  np.ascontiguousarray(elements[2], dtype=np.float64)]
            n_mat_ = self._keep[2].shape[0]
            assert el[0].shape == (n_mat_,) and el[1].shape == (n_mat_, 4) and el[2].shape == (n_mat_, 2048, 4)
            self._keep += el
            t = CTables(self._keep[1].ctypes.data_as(_dp), el[0].ctypes.data_as(_ip), el[1].ctypes.data_as(_dp),
                        el[2].ctypes.data_as(_dp))
        f = CField(field.kind, (C.c_double * 3)(*field.B), field.nr, field.nz, field.r0, field.z0, field.dr,
                   field.dz, self._keep[3].ctypes.data_as(_dp))
        n_mat = self._keep[2].shape[0]
        nbytes = lib.adept_workspace_bytes(C.byref(self.cfg), C.byref(g), n_mat, C.byref(f))
        if nbytes == 0:
            raise AdeptError(EINVAL)
        self.workspace_bytes = nbytes
        if _workspace_bytes is not None:
            nbytes = _workspace_bytes
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            ctx = C.c_void_p()
            _check(lib.adept_init(C.byref(ctx), C.byref(g), _ptr(self._keep[2]), n_mat, C.byref(t), C.byref(f),
                                  C.byref(self.cfg), C.c_void_p(self.workspace.data_ptr()), nbytes))
            self.ctx = ctx

    def close(self):
        if getattr(self, "ctx", None):
            lib.adept_shutdown(self.ctx)
            self.ctx = None

    def __del__(self):
        self.close()

    # ---- primaries
    def enqueue(self, prim, slot=0):
        """prim: dict from inputs.primaries (event, species, pos, dir, ekin); ids = index within the event."""
        ev = np.ascontiguousarray(prim["event"], dtype=np.uint32)
        n = ev.shape[0]
        first = np.r_[True, ev[1:] != ev[:-1]] if n else np.zeros(0, dtype=bool)
        start = np.maximum.accumulate(np.where(first, np.arange(n), 0)) if n else np.zeros(0, dtype=np.int64)
        ids = (np.arange(n) - start).astype(np.uint64)
        self.enqueue_batch(ev, ids, prim["species"], prim["pos"], prim["dir"], prim["ekin"], slot)

    def enqueue_batch(self, event_ids, track_ids, species, pos, direc, ekin, slot=0):
        a = [np.ascontiguousarray(event_ids, dtype=np.uint32), np.ascontiguousarray(track_ids, dtype=np.uint64),
             np.ascontiguousarray(species, dtype=np.int8), np.ascontiguousarray(pos, dtype=np.float64),
             np.ascontiguousarray(direc, dtype=np.float64), np.ascontiguousarray(ekin, dtype=np.float64)]
        _check(lib.adept_enqueue_batch(self.ctx, slot, a[0].shape[0], *[_ptr(x) for x in a]))

    def enqueue_primaries(self, slot, event_id, species, pos, direc, ekin):
        a = [np.ascontiguousarray(species, dtype=np.int8), np.ascontiguousarray(pos, dtype=np.float64),
             np.ascontiguousarray(direc, dtype=np.float64), np.ascontiguousarray(ekin, dtype=np.float64)]
        _check(lib.adept_enqueue_primaries(self.ctx, slot, event_id, a[0].shape[0], *[_ptr(x) for x in a]))

    # ---- transport
    def transport(self, slot=0, stream=None):
        _check(lib.adept_transport(self.ctx, slot, _stream_ptr(stream)))

    def transport_many(self, slots, streams):
        s = (C.c_int * len(slots))(*slots)
        p = (C.c_void_p * len(slots))(*[st.cuda_stream if hasattr(st, "cuda_stream") else int(st) for st in streams])
        _check(lib.adept_transport_many(self.ctx, len(slots), s, p))

    def read_scoring(self, slot=0, stream=None, out=None):
        edep = out if out is not None else np.zeros(self.n_volumes)
        led = CLedger()
        _check(lib.adept_read_scoring(self.ctx, slot, _ptr(edep), self.n_volumes, C.byref(led), _stream_ptr(stream)))
        return edep, led

    def read_leaked(self, slot=0, cap=1 << 16):
        out = np.zeros(cap, dtype=TRACK)
        n = C.c_size_t(0)
        _check(lib.adept_read_leaked(self.ctx, slot, _ptr(out), cap, C.byref(n)))
        return out[:min(n.value, cap)], n.value

    def stats(self, slot=0):
        s = CStats()
        _check(lib.adept_get_stats(self.ctx, slot, C.byref(s)))
        return s

    def kernel_times(self, slot=0):
        """(ms[3], launches[3]) of the gamma move / charged move / interaction kernels since the last call
        (time_kernels=1)."""
        ms = np.zeros(3)
        n = np.zeros(3, dtype=np.uint64)
        _check(lib.adept_get_kernel_times(self.ctx, slot, _ptr(ms), _ptr(n)))
        return ms, n

    def set_kernel_timing(self, on):
        _check(lib.adept_set_kernel_timing(self.ctx, 1 if on else 0))

    def raycast(self, pos, direc, navigator=NAV_BVH, max_crossings=100000, stream=None):
        """(column density [g/cm^2], boundaries crossed, kernel ms) of n rays marched through the geometry."""
        p = np.ascontiguousarray(pos, dtype=np.float64)
        d = np.ascontiguousarray(direc, dtype=np.float64)
        n = p.shape[0]
        col = np.zeros(n)
        nx = np.zeros(n, dtype=np.int32)
        ms = C.c_double(0.0)
        with self._torch.cuda.device(self.device):
            _check(lib.adept_raycast_batch(self.ctx, navigator, n, _ptr(p), _ptr(d), max_crossings, _ptr(col), _ptr(nx),
                                           C.byref(ms), _stream_ptr(stream)))
        return col, nx, ms.value

    def raycast_static(self, pos, direc, navigator=NAV_BVH, max_crossings=100000, stream=None):
        """raycast() through adept_raycast_batch_static: no device allocation, at most STATIC_MAX_RAYS rays, and
        calls that overlap on one GPU race on the library's static scratch array (include/adept.h)."""
        p = np.ascontiguousarray(pos, dtype=np.float64)
        d = np.ascontiguousarray(direc, dtype=np.float64)
        n = p.shape[0]
        col = np.zeros(n)
        nx = np.zeros(n, dtype=np.int32)
        with self._torch.cuda.device(self.device):
            _check(lib.adept_raycast_batch_static(self.ctx, navigator, n, _ptr(p), _ptr(d), max_crossings, _ptr(col), _ptr(nx),
                                                  _stream_ptr(stream)))
        return col, nx

    def iteration_trace(self, slot=0, cap=4096):
        """(t_ns[n], population[n, 3]) of the population steps since the last call (device %globaltimer;
        e-, e+, gamma tracks that entered each step)."""
        t = np.zeros(cap, dtype=np.uint64)
        pop = np.zeros((cap, 3), dtype=np.uint32)
        n = C.c_size_t(0)
        _check(lib.adept_get_iteration_trace(self.ctx, slot, _ptr(t), _ptr(pop), cap, C.byref(n)))
        return t[:n.value], pop[:n.value]

    def reset_slot(self, slot=0):
        _check(lib.adept_reset_slot(self.ctx, slot))

    # ---- test hooks
    def step_population(self, tracks, slot=0, stream=None):
        """Exactly one population step of the transport kernels on `tracks` (TRACK array, taken as given) in the
        empty slot -> TRACK array of the next population (survivors and secondaries, no particular order)."""
        tracks = np.ascontiguousarray(tracks, dtype=TRACK)
        n = tracks.shape[0]
        cap = 3 * n + 16
        out = np.zeros(cap, dtype=TRACK)
        n_out = C.c_size_t(0)
        _check(lib.adept_step_population(self.ctx, slot, n, _ptr(tracks), _ptr(out), cap, C.byref(n_out), _stream_ptr(stream)))
        assert n_out.value <= cap
        return out[:n_out.value]

    def step_frozen(self, tracks, stream=None):
        tracks = np.ascontiguousarray(tracks, dtype=TRACK)
        n = tracks.shape[0]
        res = np.zeros(n, dtype=RESULT)
        sec = np.zeros((n, 2), dtype=TRACK)
        _check(lib.adept_step_frozen(self.ctx, n, _ptr(tracks), _ptr(res), _ptr(sec), _stream_ptr(stream)))
        return res, sec

    def distance_batch(self, pos, direc, volume, s_max=None, navigator=NAV_BVH):
        pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
        direc = np.ascontiguousarray(direc, dtype=np.float64).reshape(-1, 3)
        n = pos.shape[0]
        vol = np.ascontiguousarray(np.broadcast_to(volume, (n,)), dtype=np.uint32)
        sm = np.full(n, np.inf) if s_max is None else np.ascontiguousarray(np.broadcast_to(s_max, (n,)), dtype=np.float64)
        out = np.zeros(n)
        _check(lib.adept_distance_batch(self.ctx, navigator, n, _ptr(pos), _ptr(direc), _ptr(vol), _ptr(sm), _ptr(out), None))
        return out

    def locate_batch(self, pos, navigator=NAV_BVH):
        pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
        out = np.zeros(pos.shape[0], dtype=np.int64)
        _check(lib.adept_locate_batch(self.ctx, navigator, pos.shape[0], _ptr(pos), _ptr(out), None))
        return out

    def relocate_batch(self, pos, from_volume, navigator=NAV_BVH, face=None):
        pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
        frm = np.ascontiguousarray(np.broadcast_to(from_volume, (pos.shape[0],)), dtype=np.uint32)
        fc = None if face is None else np.ascontiguousarray(np.broadcast_to(face, (pos.shape[0],)), dtype=np.int32)
        out = np.zeros(pos.shape[0], dtype=np.int64)
        _check(lib.adept_relocate_batch(self.ctx, navigator, pos.shape[0], _ptr(pos), _ptr(frm),
                                        None if fc is None else _ptr(fc), _ptr(out), None))
        return out


class HybridBuffer:
    """Host-side track buffer of the hybrid workflow: add() tracks one at a time, a batch is
    transported when `threshold` are buffered, flush() transports the rest, take() returns the accumulated
    deposits, ledger and outgoing (leaked) tracks."""

    def __init__(self, adept_obj, threshold, slot=0, stream=None):
        self._a = adept_obj
        self.h = C.c_void_p()
        _check(lib.adept_buffer_create(C.byref(self.h), adept_obj.ctx, slot, threshold, _stream_ptr(stream)))

    def add(self, event, track_id, species, pos, direc, ekin):
        p = np.ascontiguousarray(pos, dtype=np.float64)
        d = np.ascontiguousarray(direc, dtype=np.float64)
        rc = lib.adept_buffer_add(self.h, int(event), int(track_id), int(species), _ptr(p), _ptr(d), float(ekin))
        if rc < 0:
            raise AdeptError(rc)
        return rc == 1

    def flush(self):
        rc = lib.adept_buffer_flush(self.h)
        if rc < 0:
            raise AdeptError(rc)
        return rc == 1

    def pending(self):
        a, b, c = C.c_size_t(0), C.c_size_t(0), C.c_uint64(0)
        _check(lib.adept_buffer_pending(self.h, C.byref(a), C.byref(b), C.byref(c)))
        return a.value, b.value, c.value

    def take(self):
        _, n_out, _ = self.pending()
        edep = np.zeros(self._a.n_volumes)
        led = CLedger()
        out = np.zeros(max(n_out, 1), dtype=TRACK)
        n = C.c_size_t(0)
        _check(lib.adept_buffer_take(self.h, _ptr(edep), edep.shape[0], C.byref(led), _ptr(out), out.shape[0], C.byref(n)))
        return edep, led, out[:n.value]

    def close(self):
        if getattr(self, "h", None):
            lib.adept_buffer_destroy(self.h)
            self.h = None

    def __del__(self):
        self.close()
