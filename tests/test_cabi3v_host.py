"""CPU-only checks of the 3V boundary (include/landau3v.h): every declared symbol is exported and bound, the host set-up
(octree, hanging faces and edges, dof numbering, CSR pattern, integration points) -- written independently of the oracle
-- agrees with the 3V oracle bit for bit on the integer work, reproduces the paper's mesh statistics from the product
side, and compute calls refuse without a device (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2209_03228_b200 import binding as Bn
from paper_2209_03228_b200 import binding3v as B3
from paper_2209_03228_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2209_03228_b200 import build
    build.build()
    return B3.load()


@pytest.fixture(scope="module")
def o3():
    from oracle import oracle3v as O3
    O3.build()
    return O3


def test_library_exports_every_declared_3v_symbol(lib):
    text = open(os.path.join(ROOT, "include", "landau3v.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = sorted(set(re.findall(r"\b(landau3v_[a-z0-9_]+)\s*\(", text)))
    for n in ("landau3v_create", "landau3v_destroy", "landau3v_sizes", "landau3v_dof_coords", "landau3v_csr_pattern",
              "landau3v_jacobian", "landau3v_apply", "landau3v_last_error"):
        assert n in names
    assert sorted(B3.SYMBOLS) == names, "binding3v.SYMBOLS out of date with include/landau3v.h"
    for n in names:
        assert hasattr(lib, n), "liblandau_b200.so does not export %s" % n
        assert hasattr(B3, n), "binding3v lacks %s" % n


@pytest.mark.parametrize("grids", [
    [dict(half=5.0, n=4, levels=1)],                                  # the paper's grid
    [dict(half=2.0, n=3, levels=1), dict(half=1.0, n=2, levels=0)],   # odd base count: one centre cell refined
    [dict(half=3.0, n=4, levels=2)],                                  # two nested levels
    [dict(half=1.5, n=2, levels=2)],                                  # everything refined once, then the centre
])
def test_host_setup_matches_oracle(lib, o3, grids):
    species = [dict(mass=1.0, charge=-1.0, grid=g) for g in range(len(grids))]
    L = B3.Landau3V(grids, species, device=-1)
    o = o3.Oracle3V(grids, species)
    assert list(L.n_cells) == list(o.n_cells) and list(L.n_dof) == list(o.n_dof) and list(L.nnz) == list(o.nnz)
    for g in range(len(grids)):
        rp, ci = L.pattern(g)
        rp2, ci2 = o.pattern(g)
        assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)
        assert np.abs(L.dof_coords(g) - o.dof_coords(g)).max() < 1e-14 * grids[g]["half"]
        a, b = np.stack(L.ip_table(g), 1), np.stack(o.ip_table(g), 1)
        pa, pb = np.lexsort(a[:, :3].T), np.lexsort(b[:, :3].T)     # the IP order is implementation-private
        assert np.abs(a[pa] - b[pb]).max() < 1e-14 * grids[g]["half"]
    L.close()


def test_paper_mesh_statistics_from_the_product_side(lib):
    L = B3.Landau3V([dict(half=5.0, n=4, levels=1)], [dict(mass=1.0, charge=-1.0, grid=0)], device=-1)
    assert L.n_cells[0] == 120 and L.n_dof[0] == 1045 and round(L.nnz[0] / L.n_dof[0], 1) == 54.0
    L.close()


def test_no_cpu_fallback_and_argument_errors(lib):
    cfg = W.config3v("tiny")
    ctx = B3.landau3v_create(cfg["grids"], cfg["species"], cuda_device=-1)
    f = np.zeros(8)
    rc = lib.landau3v_jacobian_host(ctx, f.ctypes.data_as(C.c_void_p), C.c_int(1), C.c_double(1.0),
                                    f.ctypes.data_as(C.c_void_p), None)
    assert rc == -4 and "no CPU fallback" in B3.landau3v_last_error(ctx)
    rc = lib.landau3v_apply(ctx, f.ctypes.data_as(C.c_void_p), C.c_int(1), f.ctypes.data_as(C.c_void_p), None)
    assert rc == -4
    B3.landau3v_destroy(ctx)
    with pytest.raises(B3.LandauError):
        B3.landau3v_create([dict(half=-1.0, n=4, levels=0)], [dict(mass=1.0, charge=-1.0, grid=0)], cuda_device=-1)
    with pytest.raises(B3.LandauError):
        B3.landau3v_create([dict(half=1.0, n=4, levels=0)], [dict(mass=1.0, charge=-1.0, grid=3)], cuda_device=-1)
    with pytest.raises(B3.LandauError):
        B3.landau3v_create([dict(half=1.0, n=4, levels=0)], [dict(mass=0.0, charge=-1.0, grid=0)], cuda_device=-1)
