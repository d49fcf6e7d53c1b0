"""CPU-only checks of the product's boundary (no compute calls): the C-ABI library loads, exports every symbol
include/landau.h declares, and its host set-up (meshes, dof numbering, constraints, CSR pattern, IP tables) -- written
independently of the oracle -- agrees with the oracle's, bit for bit on the integer work."""
import os
import re

import numpy as np
import pytest

from paper_2209_03228_b200 import binding as Bn
from paper_2209_03228_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2209_03228_b200 import build
    build.build()
    return Bn.load()


def _declared_symbols(header):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(landau_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared_symbols("landau.h")
    # the calls SURVEY 8(b) lists are in the product header
    for n in ("landau_create", "landau_destroy", "landau_sizes", "landau_dof_coords", "landau_csr_pattern",
              "landau_jacobian", "landau_apply", "landau_last_error"):
        assert n in names
    debug = _declared_symbols("landau_debug.h")
    assert not set(names) & set(debug)
    for n in names + debug:
        assert hasattr(lib, n), "liblandau_b200.so does not export %s" % n
    assert sorted(Bn.SYMBOLS) == names, "binding.SYMBOLS out of date with include/landau.h"
    assert sorted(Bn.DEBUG_SYMBOLS) == debug, "binding.DEBUG_SYMBOLS out of date with include/landau_debug.h"
    for n in names + debug:  # the binding carries the same names
        assert hasattr(Bn, n), "binding lacks %s" % n


def test_reserve_refuses_without_device(lib):
    cfg = W.tiny_config("uniform", 2, batch=1)
    ctx = Bn.landau_create(cfg["grids"], cfg["species"], cfg["degree"], cuda_device=-1)
    with pytest.raises(Bn.LandauError, match="no CPU fallback"):
        Bn.landau_reserve(ctx, 4)
    with pytest.raises(Bn.LandauError):
        Bn.landau_reserve(ctx, 0)
    Bn.landau_destroy(ctx)


def test_no_cpu_fallback_compute_refuses_without_device(lib):
    cfg = W.tiny_config("uniform", 2, batch=1)
    ctx = Bn.landau_create(cfg["grids"], cfg["species"], cfg["degree"], cuda_device=-1)  # host-only context
    f = np.zeros(8)
    import ctypes as C
    rc = lib.landau_jacobian_host(ctx, f.ctypes.data_as(C.c_void_p), C.c_int(1), C.c_double(1.0),
                                  f.ctypes.data_as(C.c_void_p), None)
    assert rc == -4  # LANDAU_CUDA_ERROR: there is no CPU path behind the ABI
    assert b"no CPU fallback" in lib.landau_last_error(ctx)
    rc = lib.landau_apply_host(ctx, f.ctypes.data_as(C.c_void_p), C.c_int(1), f.ctypes.data_as(C.c_void_p), None)
    assert rc == -4
    Bn.landau_destroy(ctx)


def test_create_rejects_bad_arguments(lib):
    cfg = W.tiny_config("uniform", 2, batch=1)
    with pytest.raises(Bn.LandauError):
        Bn.landau_create(cfg["grids"], cfg["species"], 5, cuda_device=-1)               # degree unsupported
    with pytest.raises(Bn.LandauError):
        Bn.landau_create(cfg["grids"], cfg["species"], dict(degree=2, n_gauss_1d=5), cuda_device=-1)
    with pytest.raises(Bn.LandauError):
        Bn.landau_create(cfg["grids"], [dict(mass=1.0, charge=-1.0, grid=7)], 2, cuda_device=-1)
    with pytest.raises(Bn.LandauError):
        Bn.landau_create(cfg["grids"], [dict(mass=-1.0, charge=-1.0, grid=0)], 2, cuda_device=-1)


@pytest.mark.parametrize("cfg", [W.tiny_config("uniform", 2), W.tiny_config("quadtree", 3), W.tiny_config("uniform", 4),
                                 W.tiny_config("quadtree", 4), W.config(1), W.config(4), W.config(3)], ids=lambda c: c["name"])
def test_host_setup_matches_oracle(orc, lib, cfg):
    """dof numbering, CSR pattern (bit-exact), IP tables (as sets) of the product's own host set-up vs the oracle's."""
    o = orc.Oracle(cfg["grids"], cfg["species"], cfg["degree"])
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"], device=-1)
    assert list(L.n_dof) == list(o.n_dof) and list(L.nnz) == list(o.nnz)
    assert list(L.n_ip) == list(o.n_ip) and list(L.n_cells) == list(o.n_cells)
    assert L.f_stride == o.f_stride and L.csr_stride == o.v_stride
    for g in range(L.G):
        rp, ci = L.pattern(g)
        rp2, ci2 = o.pattern(g)
        assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)
        scale = cfg["grids"][g]["r_max"]
        assert np.abs(L.dof_coords(g) - o.dof_coords(g)).max() <= 1e-14 * scale
        r1, z1, w1 = L.ip_table(g)
        r2, z2, w2 = o.ip_table(g)
        p1, p2 = np.lexsort((r1, z1)), np.lexsort((r2, z2))
        assert np.abs(r1[p1] - r2[p2]).max() <= 1e-14 * scale and np.abs(z1[p1] - z2[p2]).max() <= 1e-14 * scale
        assert np.abs(w1[p1] - w2[p2]).max() <= 1e-13 * np.abs(w2).max()
    L.close()


def test_paper_mesh_statistics_from_the_product_side(lib):
    """4x2 base + one level at the origin: 14 Q3 cells, 142 equations, 22.2 nnz/row."""
    grids = [dict(kind=1, r_max=5.0, z_min=-5.0, z_max=5.0, nr=2, nz=4, levels=1)]
    L = Bn.Landau(grids, [dict(mass=1.0, charge=-1.0, grid=0)], 3, device=-1)
    assert int(L.n_cells[0]) == 14 and int(L.n_dof[0]) == 142 and int(L.nnz[0]) == 3154
    L.close()


def test_separable_detection(lib):
    cfg = W.tiny_config("uniform", 2)
    ctx = Bn.landau_create(cfg["grids"], cfg["species"], 2, cuda_device=-1)
    assert Bn.landau_is_separable(ctx)
    Bn.landau_destroy(ctx)
    ctx = Bn.landau_create(cfg["grids"], cfg["species"], 2, nu=np.array([[1.0, 2.0], [2.0, 1.0]]), cuda_device=-1)
    assert not Bn.landau_is_separable(ctx)
    Bn.landau_destroy(ctx)


@pytest.mark.parametrize("c", [1, 2, 3, 4, 5])
def test_ring_assembly_schedule_exists_for_every_baseline_config(lib, c):
    """Every BASELINE.json grid gets a shared-memory ring schedule for the assembly kernel (no gather fallback), the
    ring fits one CTA, and most CSR slots are single-contribution slots (K3)."""
    cfg = W.config(c)
    ctx = Bn.landau_create(cfg["grids"], cfg["species"], cfg["degree"], cuda_device=-1)
    sz = Bn.landau_sizes(ctx, len(cfg["grids"]))
    for g in range(len(cfg["grids"])):
        info = Bn.landau_assembly_info(ctx, g)
        assert 8 <= info["ring_cells"] <= 48           # pool of element-matrix positions, reused as matrices die
        assert info["ring_cells"] * 256 * 8 <= 220 * 1024
        assert info["n_steps"] == (int(sz["n_cells"][g]) + 7) // 8
        assert 0.7 * sz["nnz"][g] < info["n_simple_slots"] <= sz["nnz"][g]
    Bn.landau_destroy(ctx)


def test_unstructured_host_setup_matches_oracle(lib, orc):
    """landau_create_meshes (topological node identification, own bilinear geometry) against the oracle's geometric
    construction: same dofs, same pattern, same integration points and weights."""
    for k, (n, m) in ((3, (2, 2)), (2, (3, 2)), (4, (1, 2))):
        mesh = W.semicircle_mesh(5.0, n, m)
        species = [dict(mass=1.0, charge=-1.0, grid=0)]
        L = Bn.Landau.from_meshes([mesh], species, k, device=-1)
        o = orc.Oracle.from_meshes([mesh], species, k)
        assert L.n_dof[0] == o.n_dof[0] and L.nnz[0] == o.nnz[0] and L.n_ip[0] == o.n_ip[0] and L.n_cells[0] == o.n_cells[0]
        assert np.abs(L.dof_coords(0) - o.dof_coords(0)).max() < 1e-13      # same order on this mesh
        rp, ci = L.pattern(0)
        rp2, ci2 = o.pattern(0)
        assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)
        a, b = np.stack(L.ip_table(0), 1), np.stack(o.ip_table(0), 1)
        pa = np.array([int(np.argmin(((a[:, :2] - x) ** 2).sum(1))) for x in b[:, :2]])   # IP order is implementation-private
        assert len(set(pa)) == len(pa) and np.abs(a[pa] - b).max() < 1e-13
        L.close()
    # Table 13: 24 Q3 cells <-> 384 integration points, from the product side
    L = Bn.Landau.from_meshes([W.semicircle_mesh(5.0, 2, 2)], [dict(mass=1.0, charge=-1.0, grid=0)], 3, device=-1)
    assert L.n_cells[0] == 24 and L.n_ip[0] == 384
    L.close()
    v, c = W.semicircle_mesh(5.0, 2, 2)
    with pytest.raises(Bn.LandauError, match="inverted"):
        Bn.Landau.from_meshes([(v, c[:, ::-1].copy())], [dict(mass=1.0, charge=-1.0, grid=0)], 3, device=-1)
    bad = c.copy()
    bad[0, 0] = 99
    with pytest.raises(Bn.LandauError, match="missing vertex"):
        Bn.Landau.from_meshes([(v, bad)], [dict(mass=1.0, charge=-1.0, grid=0)], 3, device=-1)


@pytest.mark.parametrize("k,per_cell", [(2, 6), (3, 12), (4, 16)])
def test_triangle_host_setup_matches_oracle(lib, orc, k, per_cell):
    """Triangles P2 - P4 (landau_mesh_desc.vertices_per_cell = 3): the product's tables and topological node identification
    against the oracle's; point counts per cell as in the paper's Tables 11-12 (864/144, 816/68, 384/24)."""
    mesh = W.semicircle_triangles(5.0, 2, 2)
    species = [dict(mass=1.0, charge=-1.0, grid=0)]
    L = Bn.Landau.from_meshes([mesh], species, k, device=-1)
    o = orc.Oracle.from_meshes([mesh], species, k)
    assert L.n_ip[0] == L.n_cells[0] * per_cell == o.n_ip[0]
    assert L.n_dof[0] == o.n_dof[0] and L.nnz[0] == o.nnz[0]
    assert np.abs(L.dof_coords(0) - o.dof_coords(0)).max() < 1e-13
    rp, ci = L.pattern(0)
    rp2, ci2 = o.pattern(0)
    assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)
    a, b = np.stack(L.ip_table(0), 1), np.stack(o.ip_table(0), 1)
    pa = np.array([int(np.argmin(((a[:, :2] - x) ** 2).sum(1))) for x in b[:, :2]])
    assert len(set(pa)) == len(pa) and np.abs(a[pa] - b).max() < 1e-13
    L.close()
    quads = W.semicircle_mesh(5.0, 2, 2)
    with pytest.raises(Bn.LandauError, match="cell type"):               # one cell type per context
        Bn.Landau.from_meshes([mesh, quads], [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=2.0, charge=1.0, grid=1)], 3, device=-1)
    with pytest.raises(Bn.LandauError):                                  # Q5 quadrilaterals are not built
        Bn.Landau.from_meshes([quads], species, 5, device=-1)


def test_mesh_argument_checks(lib):
    """a one-triangle mesh (3 vertices) is a valid mesh; meshes whose coordinates are all zero or not finite
    are refused (the dof ordering divides by 2^-30 of the largest coordinate) instead of running into undefined behaviour."""
    species = [dict(mass=1.0, charge=-1.0, grid=0)]
    tri = (np.array([[0.0, -1.0], [1.5, -1.0], [0.0, 1.0]]), np.array([[0, 1, 2]], dtype=np.int32))
    L = Bn.Landau.from_meshes([tri], species, 2, device=-1)
    assert L.n_cells[0] == 1 and L.n_dof[0] == 6 and L.n_ip[0] == 6 and L.nnz[0] == 36
    L.close()
    quad3 = (tri[0], np.array([[0, 1, 2, 2]], dtype=np.int32))
    with pytest.raises(Bn.LandauError, match="fewer vertices"):
        Bn.Landau.from_meshes([quad3], species, 2, device=-1)
    for bad_value, what in ((0.0, "zero"), (float("nan"), "not finite"), (float("inf"), "not finite")):
        v = np.zeros((3, 2)) if bad_value == 0.0 else tri[0].copy()
        v[1, 0] = bad_value
        with pytest.raises(Bn.LandauError, match=what):
            Bn.Landau.from_meshes([(v, tri[1])], species, 2, device=-1)
        vq = np.zeros((4, 2)) if bad_value == 0.0 else np.array([[0.0, 0.0], [1.0, 0.0], [1.0, 1.0], [0.0, 1.0]])
        vq[2, 1] = bad_value
        with pytest.raises(Bn.LandauError, match=what):
            Bn.Landau.from_meshes([(vq, np.array([[0, 1, 2, 3]], dtype=np.int32))], species, 2, device=-1)
