"""ctypes binding of the CPU oracle (oracle/landau_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It never imports the product package and the product package never imports it.
Every function mirrors one `orc_*` entry of landau_oracle.cpp; see that file for the PAPER.md citations.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "landau_oracle.cpp")
_LIB = os.path.join(_HERE, "liblandau_oracle.so")


def build(force=False):
    """Compile the oracle with g++ -O2 -fopenmp (no tuning flags beyond that)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["g++", "-std=c++17", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


class GridDesc(C.Structure):
    _fields_ = [("kind", C.c_int), ("r_max", C.c_double), ("z_min", C.c_double), ("z_max", C.c_double),
                ("nr", C.c_int), ("nz", C.c_int), ("levels", C.c_int)]


class SpeciesDesc(C.Structure):
    _fields_ = [("mass", C.c_double), ("charge", C.c_double), ("grid", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_create.restype = C.c_void_p
        _lib.orc_tensor.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def gauss_legendre(n):
    x = np.zeros(n)
    w = np.zeros(n)
    lib().orc_gauss_legendre(C.c_int(n), _p(x), _p(w))
    return x, w


def lagrange(k, xi):
    v = np.zeros(k + 1)
    d = np.zeros(k + 1)
    lib().orc_lagrange(C.c_int(k), C.c_double(xi), _p(v), _p(d))
    return v, d


def ellip(m, mp=None):
    """{K, E, P0, P1, Dc, Q, P2} at parameter m (m' = 1-m unless given)."""
    out = np.zeros(7)
    lib().orc_ellip(C.c_double(m), C.c_double(1.0 - m if mp is None else mp), _p(out))
    return dict(zip(["K", "E", "P0", "P1", "Dc", "Q", "P2"], out))


def tensor(r, z, rb, zb):
    """Closed-form 2V tensor {UDrr, UDrz, UDzz, UKrr, UKzr} (UKrz = UDrz, UKzz = UDzz)."""
    out = np.zeros(5)
    ok = lib().orc_tensor(C.c_double(r), C.c_double(z), C.c_double(rb), C.c_double(zb), _p(out))
    return out, bool(ok)


def tensor_quadrature(r, z, rb, zb, nphi):
    """Azimuthal trapezoid rule on the 3-D tensor {UDrr, UDrz, UDzz, UKrr, UKrz, UKzr, UKzz, UDzr}."""
    out = np.zeros(8)
    lib().orc_tensor_quadrature(C.c_double(r), C.c_double(z), C.c_double(rb), C.c_double(zb), C.c_int(nphi), _p(out))
    return out


class Oracle:
    """One problem: grids + species + degree (+ optional nu matrix)."""

    def __init__(self, grids, species, degree, nu=None, threads=None):
        """grids: list of dicts(kind,r_max,z_min,z_max,nr,nz,levels); species: list of dicts(mass,charge,grid)."""
        L = lib()
        self.G = len(grids)
        self.S = len(species)
        self.degree = degree
        self.species = [dict(s) for s in species]
        self.grids = [dict(g) for g in grids]
        g_arr = (GridDesc * self.G)(*[GridDesc(int(g["kind"]), float(g["r_max"]), float(g["z_min"]), float(g["z_max"]),
                                              int(g["nr"]), int(g["nz"]), int(g.get("levels", 0))) for g in grids])
        s_arr = (SpeciesDesc * self.S)(*[SpeciesDesc(float(s["mass"]), float(s["charge"]), int(s["grid"]))
                                         for s in species])
        self.threads = int(threads) if threads else (os.cpu_count() or 1)
        nu_p = None
        if nu is not None:
            self._nu = np.ascontiguousarray(nu, dtype=np.float64)
            nu_p = _p(self._nu)
        self.h = C.c_void_p(L.orc_create(g_arr, C.c_int(self.G), s_arr, C.c_int(self.S), C.c_int(degree), nu_p,
                                         C.c_int(self.threads)))
        self._sizes(species)

    def _sizes(self, species):
        L = lib()
        n_dof = np.zeros(self.G, np.int32)
        nnz = np.zeros(self.G, np.int32)
        n_ip = np.zeros(self.G, np.int32)
        n_cells = np.zeros(self.G, np.int32)
        fs = C.c_longlong()
        vs = C.c_longlong()
        L.orc_sizes(self.h, _p(n_dof), _p(nnz), _p(n_ip), _p(n_cells), C.byref(fs), C.byref(vs))
        self.n_dof, self.nnz, self.n_ip, self.n_cells = n_dof, nnz, n_ip, n_cells
        self.f_stride, self.v_stride = fs.value, vs.value
        self.sgrid = [int(s["grid"]) for s in species]
        self.f_off = np.concatenate([[0], np.cumsum([n_dof[g] for g in self.sgrid])]).astype(np.int64)
        self.v_off = np.concatenate([[0], np.cumsum([nnz[g] for g in self.sgrid])]).astype(np.int64)
        self.ip_off = np.concatenate([[0], np.cumsum([n_ip[g] for g in self.sgrid])]).astype(np.int64)

    @classmethod
    def from_meshes(cls, meshes, species, degree, nu=None, threads=None):
        """Unstructured grids: meshes = list of (vertices [nv, 2] (r, z), cells [nc, 4] or [nc, 3] counter-clockwise)."""
        self = cls.__new__(cls)
        L = lib()
        L.orc_create_meshes.restype = C.c_void_p
        self.G, self.S, self.degree = len(meshes), len(species), degree
        self.species = [dict(s) for s in species]
        self.grids = [dict(kind=2) for _ in meshes]
        self._v = [np.ascontiguousarray(m[0], dtype=np.float64) for m in meshes]
        self._c = [np.ascontiguousarray(m[1], dtype=np.int32) for m in meshes]
        nv = np.array([len(v) for v in self._v], dtype=np.int32)
        nc = np.array([len(c) for c in self._c], dtype=np.int32)
        vp = (C.c_void_p * self.G)(*[v.ctypes.data for v in self._v])
        cp = (C.c_void_p * self.G)(*[c.ctypes.data for c in self._c])
        s_arr = (SpeciesDesc * self.S)(*[SpeciesDesc(float(s["mass"]), float(s["charge"]), int(s["grid"])) for s in species])
        self.threads = int(threads) if threads else (os.cpu_count() or 1)
        nu_p = None
        if nu is not None:
            self._nu = np.ascontiguousarray(nu, dtype=np.float64)
            nu_p = _p(self._nu)
        vpc = int(self._c[0].shape[1])
        assert all(c.shape[1] == vpc for c in self._c)
        h = L.orc_create_meshes(C.c_int(self.G), _p(nv), vp, _p(nc), cp, C.c_int(vpc), s_arr, C.c_int(self.S), C.c_int(degree),
                                nu_p, C.c_int(self.threads))
        if not h:
            raise RuntimeError("orc_create_meshes failed (inverted cell)")
        self.h = C.c_void_p(h)
        self._sizes(species)
        return self

    def __del__(self):
        try:
            lib().orc_destroy(self.h)
        except Exception:
            pass

    def dof_coords(self, g):
        rz = np.zeros((self.n_dof[g], 2))
        lib().orc_dof_coords(self.h, C.c_int(g), _p(rz))
        return rz

    def pattern(self, g):
        rp = np.zeros(self.n_dof[g] + 1, np.int32)
        ci = np.zeros(self.nnz[g], np.int32)
        lib().orc_pattern(self.h, C.c_int(g), _p(rp), _p(ci))
        return rp, ci

    def ip_table(self, g):
        r = np.zeros(self.n_ip[g])
        z = np.zeros(self.n_ip[g])
        w = np.zeros(self.n_ip[g])
        lib().orc_ip_table(self.h, C.c_int(g), _p(r), _p(z), _p(w))
        return r, z, w

    def cells(self, g):
        rect = np.zeros((self.n_cells[g], 4))
        lib().orc_cells(self.h, C.c_int(g), _p(rect))
        return rect

    def fields(self, fentry, s):
        fentry = np.ascontiguousarray(fentry, dtype=np.float64)
        n = self.n_ip[self.sgrid[s]]
        f, fr, fz = np.zeros(n), np.zeros(n), np.zeros(n)
        lib().orc_fields(self.h, _p(fentry), C.c_int(s), _p(f), _p(fr), _p(fz))
        return f, fr, fz

    def inner(self, fentry):
        """list over species of [n_ip, 5] arrays (Drr, Drz, Dzz, Kr, Kz)."""
        fentry = np.ascontiguousarray(fentry, dtype=np.float64)
        assert fentry.size == self.f_stride
        out = np.zeros(int(self.ip_off[-1]) * 5)
        lib().orc_inner(self.h, _p(fentry), _p(out))
        return [out[5 * self.ip_off[s]:5 * self.ip_off[s + 1]].reshape(-1, 5) for s in range(self.S)]

    def inner_at_points(self, alpha, fsrc, rz):
        """D,K of species alpha at free field points rz[npts,2]; fsrc[beta] = [n_ip,3] analytic samples."""
        rz = np.ascontiguousarray(rz, dtype=np.float64)
        arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in fsrc]
        ptrs = (C.c_void_p * self.S)(*[a.ctypes.data for a in arrs])
        out = np.zeros((rz.shape[0], 5))
        lib().orc_inner_at_points(self.h, C.c_int(alpha), ptrs, _p(rz), C.c_int(rz.shape[0]), _p(out))
        return out

    def jacobian(self, fentry, dt):
        fentry = np.ascontiguousarray(fentry, dtype=np.float64)
        assert fentry.size == self.f_stride
        vals = np.zeros(self.v_stride)
        lib().orc_jacobian(self.h, _p(fentry), C.c_double(dt), _p(vals))
        return vals

    def apply(self, fentry):
        fentry = np.ascontiguousarray(fentry, dtype=np.float64)
        assert fentry.size == self.f_stride
        rhs = np.zeros(self.f_stride)
        lib().orc_apply(self.h, _p(fentry), _p(rhs))
        return rhs

    def mass(self, g):
        vals = np.zeros(self.nnz[g])
        lib().orc_mass(self.h, C.c_int(g), _p(vals))
        return vals

    # batch conveniences: plain loops over entries (entries are independent)
    def jacobian_batch(self, batch_f, dt):
        return np.stack([self.jacobian(f, dt) for f in np.asarray(batch_f).reshape(-1, self.f_stride)])

    def apply_batch(self, batch_f):
        return np.stack([self.apply(f) for f in np.asarray(batch_f).reshape(-1, self.f_stride)])
