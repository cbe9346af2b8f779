"""The C-ABI library loads without a GPU and exports every symbol include/rt.h declares; the host-side
argument checks that need no device answer with error codes, not exceptions.  CPU only."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "rt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rt_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for n in ("rt_create", "rt_workspace_bytes", "rt_mesh_upload", "rt_state_init", "rt_step", "rt_download",
              "rt_last_error", "rt_destroy"):
        assert n in names


def test_library_exports_every_declared_symbol():
    from paper_2404_17630_b200.build import build_rt
    L = ctypes.CDLL(build_rt())
    for n in declared_functions():
        assert hasattr(L, n), n


def test_binding_has_the_same_names():
    from paper_2404_17630_b200 import rt
    for n in ("rt_create", "rt_workspace_bytes", "rt_mesh_upload", "rt_state_init", "rt_step", "rt_download",
              "rt_last_error", "rt_destroy"):
        assert callable(getattr(rt, n))


def test_workspace_bytes_and_null_arguments_need_no_device():
    from paper_2404_17630_b200 import rt
    L = rt.lib()
    assert rt.rt_workspace_bytes(0, 10, 1) == 0
    assert rt.rt_workspace_bytes(10, 10, 9) == 0
    small, big = rt.rt_workspace_bytes(10 ** 6, 3 * 10 ** 6, 1), rt.rt_workspace_bytes(10 ** 6, 3 * 10 ** 6, 8)
    assert 0 < small < big
    # config 4 (384^3 cells, 7.72 faces per cell, 3 groups) must fit the 180 GB of one B200
    assert rt.rt_workspace_bytes(384 ** 3, int(7.72 * 384 ** 3), 3) < 150e9
    assert L.rt_step(None, 1.0, 1) == -1          # RT_EINVAL, no abort
    assert L.rt_download(None, None, None) == -1
    assert L.rt_last_error(None) == b"null context"
    L.rt_destroy(None)


def test_every_north_star_call_cites_its_passage():
    """Each of the eight calls of SURVEY 8(b) carries, in the comment right above its declaration, the
    PAPER.md passage (or the SURVEY convention) that defines it."""
    src = open(os.path.join(ROOT, "include", "rt.h")).read()
    for n in ("rt_create", "rt_workspace_bytes", "rt_mesh_upload", "rt_state_init", "rt_step", "rt_download",
              "rt_last_error", "rt_destroy"):
        m = re.search(r"/\*((?:(?!\*/).)*)\*/\s*(?:const\s+char|size_t|int|void)\s*\*?\s*%s\s*\(" % n, src, flags=re.S)
        assert m, n
        assert re.search(r"PAPER\.md:\d+|SURVEY 8\(b\)", m.group(1)), n


def test_the_library_reads_no_environment_variable():
    csrc = os.path.join(ROOT, "paper_2404_17630_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f
    assert "environ" not in open(os.path.join(ROOT, "paper_2404_17630_b200", "rt.py")).read()


def test_tuning_struct_matches_the_header():
    from paper_2404_17630_b200 import rt
    assert ctypes.sizeof(rt.rt_tuning) == 4 * (7 + 6 + 1 + 9)
    L = rt.lib()
    assert L.rt_set_tuning(None, None) == -1


def test_new_entry_points_answer_without_a_device():
    """Sharded-run calls with a null context, and the no-allocation call's size check, return error codes on a
    machine without a GPU: no abort, no exception."""
    from paper_2404_17630_b200 import rt
    L = rt.lib()
    L.rt_step_phase.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.c_int]
    assert L.rt_step_phase(None, 1.0, 0) == -1
    L.rt_halo_pack.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
    L.rt_halo_unpack.argtypes = L.rt_halo_pack.argtypes
    assert L.rt_halo_pack(None, 0, 0, None, None) == -1 and L.rt_halo_unpack(None, 1, 0, None, None) == -1
    L.rt_halo_row_bytes.argtypes = [ctypes.c_void_p, ctypes.c_int]
    assert L.rt_halo_row_bytes(None, 0) == -1
    L.rt_stored_photons_noalloc.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_void_p,
                                            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_char_p, ctypes.c_int]
    err = ctypes.create_string_buffer(256)
    assert L.rt_stored_photons_noalloc(0, None, rt.RT_NOALLOC_MAX_CELLS + 1, 1, None, None, None, err, 256) == -1
    assert b"RT_NOALLOC_MAX_CELLS" in err.value
    assert L.rt_stored_photons_noalloc(0, None, 10, 0, None, None, None, err, 256) == -1 and b"ngroup" in err.value
    src = open(os.path.join(ROOT, "include", "rt.h")).read()
    assert "#define RT_NOALLOC_MAX_CELLS (1 << 24)" in src and rt.RT_NOALLOC_MAX_CELLS == 1 << 24
    assert (rt.RT_PHASE_CHEM, rt.RT_PHASE_GRAD1, rt.RT_PHASE_FLUX1, rt.RT_PHASE_GRAD2, rt.RT_PHASE_FLUX2) == (0, 1, 2, 3, 4)
    assert "enum { RT_PHASE_CHEM = 0, RT_PHASE_GRAD1 = 1, RT_PHASE_FLUX1 = 2, RT_PHASE_GRAD2 = 3, RT_PHASE_FLUX2 = 4 };" in src
