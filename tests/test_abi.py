"""The C-ABI library loads and exports every symbol include/dd4dvar.h declares (no compute)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2205_06649_b200 import build
    return ctypes.CDLL(build.build())


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "dd4dvar.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dd4dvar_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = declared_symbols()
    for n in ("dd4dvar_create", "dd4dvar_set_background", "dd4dvar_set_observations", "dd4dvar_run",
              "dd4dvar_eval_local", "dd4dvar_eval_global"):
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    for n in declared_symbols():
        assert hasattr(lib, n), n


def test_binding_lists_the_same_symbols(lib):
    from paper_2205_06649_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()


def test_create_rejects_bad_arguments_without_a_gpu(lib):
    from paper_2205_06649_b200.binding import Grid, Decomp, Window, Opts
    lib.dd4dvar_create.argtypes = [ctypes.c_void_p] * 6
    h = ctypes.c_void_p()
    g = Grid(36, 18, 6.371e6, 7.292e-5, 9.806, 0.64, 0.02)
    w = Window(600.0, 16)
    o = Opts(5, 5, 20, 1e-4, 0)
    # more windows than steps, tile rows without room for the ghost ring: -2 (does not fit)
    for d in (Decomp(2, 2, 17, 1, 1.0, 1.0), Decomp(2, 9, 2, 1, 1.0, 1.0)):
        rc = lib.dd4dvar_create(ctypes.byref(g), ctypes.byref(d), ctypes.byref(w), ctypes.byref(o), None, ctypes.byref(h))
        assert rc == -2 and not h.value
    bad = Grid(2, 18, 6.371e6, 7.292e-5, 9.806, 0.64, 0.02)
    d = Decomp(1, 1, 1, 0, 1.0, 1.0)
    assert lib.dd4dvar_create(ctypes.byref(bad), ctypes.byref(d), ctypes.byref(w), ctypes.byref(o), None, ctypes.byref(h)) == -1
    # a valid layout builds its geometry on the host and reports sizes without touching a device
    d = Decomp(2, 2, 2, 1, 1.0, 1.0)
    assert lib.dd4dvar_create(ctypes.byref(g), ctypes.byref(d), ctypes.byref(w), ctypes.byref(o), None, ctypes.byref(h)) == 0
    lib.dd4dvar_num_subdomains.argtypes = [ctypes.c_void_p]
    lib.dd4dvar_workspace_bytes.argtypes = [ctypes.c_void_p]
    lib.dd4dvar_workspace_bytes.restype = ctypes.c_size_t
    assert lib.dd4dvar_num_subdomains(h) == 8
    assert lib.dd4dvar_workspace_bytes(h) > 0
    out = (ctypes.c_int * 16)()
    lib.dd4dvar_subdomain_info.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
    assert lib.dd4dvar_subdomain_info(h, 3, out) == 0
    # tile (1,1) of window 0: owned 18..36 x 9..18, extended by 1 cell on interior sides (eq (70))
    assert list(out)[:11] == [1, 1, 0, 18, 36, 9, 18, 17, 8, 20, 10]
    lib.dd4dvar_destroy.argtypes = [ctypes.c_void_p]
    lib.dd4dvar_destroy(h)


def test_geometry_matches_oracle_on_ragged_layouts(lib):
    from oracle import Oracle
    from paper_2205_06649_b200.binding import Grid, Decomp, Window, Opts
    lib.dd4dvar_create.argtypes = [ctypes.c_void_p] * 6
    lib.dd4dvar_subdomain_info.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
    lib.dd4dvar_num_subdomains.argtypes = [ctypes.c_void_p]
    lib.dd4dvar_destroy.argtypes = [ctypes.c_void_p]
    for (nlon, nlat, N, p1, p2, q, o) in [(36, 18, 16, 2, 2, 2, 1), (40, 23, 17, 3, 2, 3, 2), (36, 18, 16, 1, 1, 1, 0),
                                          (48, 30, 10, 1, 3, 2, 2), (720, 360, 128, 16, 16, 8, 2)]:
        h = ctypes.c_void_p()
        g = Grid(nlon, nlat, 6.371e6, 7.292e-5, 9.806, 0.64, 0.02)
        d = Decomp(p1, p2, q, o, 1.0, 1.0); w = Window(100.0, N); op = Opts(5, 5, 20, 1e-4, 0)
        assert lib.dd4dvar_create(ctypes.byref(g), ctypes.byref(d), ctypes.byref(w), ctypes.byref(op), None, ctypes.byref(h)) == 0
        orc = Oracle(nlon, nlat, 100.0, N, p1, p2, q, o)
        assert lib.dd4dvar_num_subdomains(h) == orc.nsub
        for k in range(orc.nsub):
            out = (ctypes.c_int * 16)()
            lib.dd4dvar_subdomain_info(h, k, out)
            assert list(out) == [orc.subs[k][f] for f in ("a", "b", "jw", "oi0", "oi1", "oj0", "oj1", "ei0", "ej0",
                                                           "ex", "ey", "gx", "gys", "gyn", "s", "e")], k
        lib.dd4dvar_destroy(h)


def test_geometry_follows_the_definitions_written_out_in_python(lib):
    """Third statement of the decomposition, from the text and independent of both C codes: Def 3
    and eq (70) (l.1024) with the ragged split of DESIGN.md R9.  Tile a owns the columns floor(a nlon / p1) ..
    floor((a+1) nlon / p1) - 1 (rows alike), the extended tile adds `o` cells on every side that has a neighbour
    (longitude is periodic: both sides whenever p1 > 1; latitude ends at the poles), the frozen ghost ring is 3 cells
    wide wherever the extended tile has a neighbour, window j covers the steps floor(j N / q) .. floor((j+1) N / q)."""
    from paper_2205_06649_b200.binding import Grid, Decomp, Window, Opts
    lib.dd4dvar_create.argtypes = [ctypes.c_void_p] * 6
    lib.dd4dvar_subdomain_info.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
    lib.dd4dvar_num_subdomains.argtypes = [ctypes.c_void_p]
    lib.dd4dvar_destroy.argtypes = [ctypes.c_void_p]
    for (nlon, nlat, N, p1, p2, q, o) in [(36, 18, 16, 2, 2, 2, 1), (40, 23, 17, 3, 2, 3, 2), (36, 18, 16, 1, 1, 1, 0),
                                          (48, 30, 10, 1, 3, 2, 2), (50, 31, 9, 5, 4, 3, 1), (1440, 720, 256, 16, 16, 8, 2)]:
        h = ctypes.c_void_p()
        g = Grid(nlon, nlat, 6.371e6, 7.292e-5, 9.806, 0.64, 0.02)
        d = Decomp(p1, p2, q, o, 1.0, 1.0); w = Window(100.0, N); op = Opts(5, 5, 20, 1e-4, 0)
        assert lib.dd4dvar_create(ctypes.byref(g), ctypes.byref(d), ctypes.byref(w), ctypes.byref(op), None, ctypes.byref(h)) == 0
        assert lib.dd4dvar_num_subdomains(h) == p1 * p2 * q
        covered = np.zeros((q, nlat, nlon), dtype=int)
        for jw in range(q):
            for b in range(p2):
                for a in range(p1):
                    k = (jw * p2 + b) * p1 + a
                    out = (ctypes.c_int * 16)()
                    lib.dd4dvar_subdomain_info(h, k, out)
                    own_i = list(range((a * nlon) // p1, ((a + 1) * nlon) // p1))     # R9: boundaries at floor(a n / p)
                    own_j = list(range((b * nlat) // p2, ((b + 1) * nlat) // p2))
                    ext_i = list(range(own_i[0] - o, own_i[-1] + o + 1)) if p1 > 1 else own_i
                    ext_j = [j for j in range(own_j[0] - o, own_j[-1] + o + 1) if 0 <= j < nlat] if p2 > 1 else own_j
                    steps = list(range((jw * N) // q, ((jw + 1) * N) // q))         # steps of window jw
                    want = [a, b, jw, own_i[0], own_i[-1] + 1, own_j[0], own_j[-1] + 1, ext_i[0], ext_j[0],
                            len(ext_i), len(ext_j), 3 if p1 > 1 else 0, 3 if ext_j[0] > 0 else 0,
                            3 if ext_j[-1] < nlat - 1 else 0, steps[0], steps[-1] + 1]
                    assert list(out) == want, (k, list(out), want)
                    covered[jw][np.ix_(own_j, own_i)] += 1
        assert np.all(covered == 1)             # the owned tiles partition the grid in every window
        lib.dd4dvar_destroy(h)


def test_wavefront_kernels_take_layouts_up_to_their_row_limit_and_no_further(lib):
    """Eligibility of the wavefront kernels: the resident state has a compile-time number of rows
    (80 for tiles of up to 68 padded columns, 49 up to 100).  One row more: the default falls back to another kernel
    family and an explicit request for the wavefront path is refused (-2), without a GPU."""
    from paper_2205_06649_b200.binding import Grid, Decomp, Window, Opts
    lib.dd4dvar_create.argtypes = [ctypes.c_void_p] * 6
    lib.dd4dvar_active_path.argtypes = [ctypes.c_void_p]
    lib.dd4dvar_destroy.argtypes = [ctypes.c_void_p]

    def create(nlon, nlat, path):
        h = ctypes.c_void_p()
        g = Grid(nlon, nlat, 6.371e6, 7.292e-5, 9.806, 0.64, 0.02)
        d = Decomp(2, 2, 2, 2, 1.0, 1.0); w = Window(60.0, 8); op = Opts(5, 5, 20, 1e-4, path)
        rc = lib.dd4dvar_create(ctypes.byref(g), ctypes.byref(d), ctypes.byref(w), ctypes.byref(op), None, ctypes.byref(h))
        p = lib.dd4dvar_active_path(h) if rc == 0 else None
        if rc == 0:
            lib.dd4dvar_destroy(h)
        return rc, p

    assert create(116, 156, 0) == (0, 5)            # extended tiles 62 x 80 (K = 2)
    assert create(116, 158, 0)[1] in (1, 2)         # 62 x 81
    assert create(116, 158, 5)[0] == -2
    assert create(180, 94, 0) == (0, 5)             # 94 x 49 (K = 3)
    assert create(180, 96, 0)[1] in (1, 2)          # 94 x 50
    assert create(180, 96, 5)[0] == -2
