"""The C-ABI library loads and exports every symbol include/adept.h declares (no compute, no GPU)."""
import ctypes as C
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "adept.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(adept_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = declared_symbols()
    for must in ("adept_init", "adept_enqueue_primaries", "adept_transport", "adept_read_scoring",
                 "adept_workspace_bytes", "adept_read_leaked", "adept_get_stats", "adept_step_frozen", "adept_shutdown"):
        assert must in names


def test_library_exports_every_declared_symbol():
    import __graft_entry__
    __graft_entry__.build()
    lib = C.CDLL(os.path.join(ROOT, "paper_2209_15445_b200", "libadept_b200.so"))
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_binding_structs_match_the_header_layout():
    from paper_2209_15445_b200 import adept
    # sizes as a C compiler sees include/adept.h
    import subprocess
    import tempfile
    with tempfile.TemporaryDirectory() as tmp:
        src = os.path.join(tmp, "sz.c")
        open(src, "w").write('#include <stdio.h>\n#include "adept.h"\nint main(void){printf("%zu %zu %zu %zu %zu %zu %zu\\n",'
                             'sizeof(adept_config),sizeof(adept_stats),sizeof(adept_ledger),sizeof(adept_track),'
                             'sizeof(adept_step_result),sizeof(adept_geometry),sizeof(adept_field));return 0;}\n')
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", os.path.join(tmp, "sz"), src])
        sizes = [int(x) for x in subprocess.check_output([os.path.join(tmp, "sz")]).split()]
    assert sizes == [C.sizeof(adept.CConfig), C.sizeof(adept.CStats), C.sizeof(adept.CLedger), adept.TRACK.itemsize,
                     adept.RESULT.itemsize, C.sizeof(adept.CGeometry), C.sizeof(adept.CField)]
    assert C.sizeof(adept.CConfig) == 120 and C.sizeof(adept.CStats) == 184 and C.sizeof(adept.CLedger) == 40
    assert adept.TRACK.itemsize == 80 and adept.RESULT.itemsize == 136
    cfg = adept.default_config()
    assert cfg.delta_chord == 1e-3 and cfg.eps_push == 1e-7 and cfg.chord_budget == 16 and cfg.navigator == adept.NAV_BVH
    assert set(adept.EXPORTS) == set(declared_symbols())


def test_invalid_arguments_are_reported_without_a_gpu():
    from paper_2209_15445_b200 import adept
    assert adept.lib.adept_workspace_bytes(None, None, 0, None) == 0
    assert b"null" in adept.lib.adept_last_error()
    assert adept.lib.adept_transport(None, 0, None) == adept.EINVAL
    assert adept.lib.adept_shutdown(None) == adept.EINVAL


def test_workspace_size_accounts_for_tracks_and_bvh(calo):
    from paper_2209_15445_b200 import adept
    from paper_2209_15445_b200.inputs import field
    g, mats, tabs, scal = calo
    f = field.no_field()
    cg = adept.CGeometry(g.n_volumes, g.solid.ctypes.data_as(adept._ip), g.dims.ctypes.data_as(adept._dp),
                         g.material.ctypes.data_as(adept._ip), g.mother.ctypes.data_as(adept._ip),
                         g.daughter_begin.ctypes.data_as(adept._ip), g.daughter_count.ctypes.data_as(adept._ip),
                         g.rot.ctypes.data_as(adept._dp), g.trans.ctypes.data_as(adept._dp))
    cf = adept.CField(f.kind, (C.c_double * 3)(*f.B), 0, 0, 0, 0, 1, 1, None)
    small = adept.lib.adept_workspace_bytes(C.byref(adept.default_config(track_capacity=1 << 10)), C.byref(cg), 3, C.byref(cf))
    big = adept.lib.adept_workspace_bytes(C.byref(adept.default_config(track_capacity=1 << 12)), C.byref(cg), 3, C.byref(cf))
    assert small > 0 and big - small >= 3 * 1024 * 6 * 76          # 2 buffers x 3 species x 76 B per extra track
    two = adept.lib.adept_workspace_bytes(C.byref(adept.default_config(track_capacity=1 << 10, n_event_slots=2)), C.byref(cg), 3, C.byref(cf))
    assert two > small
    bad = adept.default_config(track_capacity=1)
    assert adept.lib.adept_workspace_bytes(C.byref(bad), C.byref(cg), 3, C.byref(cf)) == 0
