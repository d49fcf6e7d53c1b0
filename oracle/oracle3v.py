"""ctypes binding of the 3V CPU oracle (oracle/landau3v_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.  It never
imports the product package and the product package never imports it.  Every function mirrors one `orc3_*` entry of
landau3v_oracle.cpp; see that file for the PAPER.md citations.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "landau3v_oracle.cpp")
_LIB = os.path.join(_HERE, "liblandau3v_oracle.so")


def build(force=False):
    """Compile the oracle with g++ -O2 -fopenmp (no tuning flags beyond that)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc3_create.restype = C.c_void_p
        _lib.orc3_threads.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def tensor(v, vb):
    """Landau tensor U(v, vb) as (xx, xy, xz, yy, yz, zz); zeros for coincident points."""
    v = np.ascontiguousarray(v, dtype=np.float64)
    vb = np.ascontiguousarray(vb, dtype=np.float64)
    out = np.zeros(6)
    lib().orc3_tensor(_p(v), _p(vb), _p(out))
    return out


class Oracle3V:
    """One 3V problem.  grids: list of dicts(half, n, levels): Q2 hexahedra on [-half, half]^3, n^3 base cells, `levels`
    refinements of the cells touching the origin; species: list of dicts(mass, charge, grid)."""

    def __init__(self, grids, species, nu=None):
        L = lib()
        self.G, self.S = len(grids), len(species)
        self.grids = [dict(g) for g in grids]
        self.species = [dict(s) for s in species]
        half = np.array([g["half"] for g in grids], dtype=np.float64)
        n = np.array([g["n"] for g in grids], dtype=np.int32)
        lev = np.array([g.get("levels", 0) for g in grids], dtype=np.int32)
        mass = np.array([s["mass"] for s in species], dtype=np.float64)
        charge = np.array([s["charge"] for s in species], dtype=np.float64)
        grid = np.array([s["grid"] for s in species], dtype=np.int32)
        nu_p = None
        if nu is not None:
            self._nu = np.ascontiguousarray(nu, dtype=np.float64)
            nu_p = _p(self._nu)
        h = L.orc3_create(C.c_int(self.G), _p(half), _p(n), _p(lev), C.c_int(self.S), _p(mass), _p(charge), _p(grid), nu_p)
        if not h:
            raise RuntimeError("orc3_create failed (unresolvable constraints)")
        self.h = C.c_void_p(h)
        self.threads = int(L.orc3_threads())
        n_dof, nnz, n_ip, n_cells = (np.zeros(self.G, np.int32) for _ in range(4))
        L.orc3_sizes(self.h, _p(n_dof), _p(nnz), _p(n_ip), _p(n_cells))
        self.n_dof, self.nnz, self.n_ip, self.n_cells = n_dof, nnz, n_ip, n_cells
        self.sgrid = [int(s["grid"]) for s in species]
        self.f_off = np.concatenate([[0], np.cumsum([n_dof[g] for g in self.sgrid])]).astype(np.int64)
        self.v_off = np.concatenate([[0], np.cumsum([nnz[g] for g in self.sgrid])]).astype(np.int64)
        self.ip_off = np.concatenate([[0], np.cumsum([n_ip[g] for g in self.sgrid])]).astype(np.int64)
        self.f_stride, self.v_stride = int(self.f_off[-1]), int(self.v_off[-1])

    def __del__(self):
        try:
            lib().orc3_destroy(self.h)
        except Exception:
            pass

    def dof_coords(self, g):
        xyz = np.zeros((self.n_dof[g], 3))
        lib().orc3_dof_coords(self.h, C.c_int(g), _p(xyz))
        return xyz

    def pattern(self, g):
        rp = np.zeros(self.n_dof[g] + 1, np.int32)
        ci = np.zeros(self.nnz[g], np.int32)
        lib().orc3_pattern(self.h, C.c_int(g), _p(rp), _p(ci))
        return rp, ci

    def ip_table(self, g):
        x, y, z, w = (np.zeros(self.n_ip[g]) for _ in range(4))
        lib().orc3_ip_table(self.h, C.c_int(g), _p(x), _p(y), _p(z), _p(w))
        return x, y, z, w

    def fields(self, fentry, s):
        """[n_ip, 4]: f and its gradient at the integration points of species s."""
        fentry = np.ascontiguousarray(fentry, dtype=np.float64)
        out = np.zeros((self.n_ip[self.sgrid[s]], 4))
        lib().orc3_fields(self.h, _p(fentry), C.c_int(s), _p(out))
        return out

    def inner(self, fentry):
        """list over species of [n_ip, 9] arrays (Dxx, Dxy, Dxz, Dyy, Dyz, Dzz, Kx, Ky, Kz)."""
        fentry = np.ascontiguousarray(fentry, dtype=np.float64)
        assert fentry.size == self.f_stride
        out = np.zeros(int(self.ip_off[-1]) * 9)
        lib().orc3_inner(self.h, _p(fentry), _p(out))
        return [out[9 * self.ip_off[s]:9 * self.ip_off[s + 1]].reshape(-1, 9) for s in range(self.S)]

    def inner_at_points(self, alpha, fsrc, pts):
        """D, K of species alpha at free field points pts[npts, 3]; fsrc[beta] = [n_ip, 4] samples of f, grad f."""
        pts = np.ascontiguousarray(pts, dtype=np.float64)
        arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in fsrc]
        ptrs = (C.c_void_p * self.S)(*[a.ctypes.data for a in arrs])
        out = np.zeros((pts.shape[0], 9))
        lib().orc3_inner_at_points(self.h, C.c_int(alpha), ptrs, _p(pts), C.c_int(pts.shape[0]), _p(out))
        return out

    def jacobian(self, fentry, dt):
        fentry = np.ascontiguousarray(fentry, dtype=np.float64)
        assert fentry.size == self.f_stride
        vals = np.zeros(self.v_stride)
        lib().orc3_jacobian(self.h, _p(fentry), C.c_double(dt), _p(vals))
        return vals

    def apply(self, fentry):
        fentry = np.ascontiguousarray(fentry, dtype=np.float64)
        assert fentry.size == self.f_stride
        rhs = np.zeros(self.f_stride)
        lib().orc3_apply(self.h, _p(fentry), _p(rhs))
        return rhs

    def mass(self, g):
        vals = np.zeros(self.nnz[g])
        lib().orc3_mass(self.h, C.c_int(g), _p(vals))
        return vals

    def jacobian_batch(self, batch_f, dt):
        return np.stack([self.jacobian(f, dt) for f in np.asarray(batch_f).reshape(-1, self.f_stride)])

    def apply_batch(self, batch_f):
        return np.stack([self.apply(f) for f in np.asarray(batch_f).reshape(-1, self.f_stride)])
