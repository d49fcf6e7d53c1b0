"""Thin ctypes binding of include/landau.h (argument marshalling only -- every step runs in the CUDA kernels).

Functions carry the C names (landau_create, landau_jacobian, landau_apply, ...).  PyTorch is used by callers for
device memory and streams only; tensors are passed as raw device pointers.  There is no CPU fallback: if the
shared library is missing or cannot be loaded, `load()` raises, and every entry point goes through `load()`.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblandau_b200.so")

LANDAU_OK = 0
STATUS = {0: "LANDAU_OK", -1: "LANDAU_INVALID_ARG", -2: "LANDAU_UNSUPPORTED", -3: "LANDAU_OUT_OF_MEMORY",
          -4: "LANDAU_CUDA_ERROR", -5: "LANDAU_NOT_CONVERGED"}
LANDAU_NOT_CONVERGED = -5

# every symbol include/landau.h (the product ABI) and include/landau_debug.h (diagnostics, probes, tuning knobs)
# declare; tests check that the headers and these lists agree and that the library exports all of them
SYMBOLS = ["landau_create", "landau_create_meshes", "landau_destroy", "landau_sizes", "landau_dof_coords", "landau_ip_table",
           "landau_csr_pattern", "landau_csr_pattern_host", "landau_jacobian", "landau_apply", "landau_spmv",
           "landau_solve", "landau_solve_noalloc", "landau_jacobian_apply", "landau_step", "landau_jacobian_host", "landau_apply_host",
           "landau_reserve", "landau_last_error"]
DEBUG_SYMBOLS = ["landau_last_coefficients", "landau_tensor_eval", "landau_ellip_eval", "landau_fp64_probe", "landau_l2_probe",
                 "landau_launch_count", "landau_is_separable", "landau_set_timing", "landau_last_stage_ms",
                 "landau_set_inner_kernel", "landau_set_assembly_kernel", "landau_set_solve_kernel", "landau_solve_mode", "landau_assembly_info",
                 "landau_set_batch_chunk"]


class LandauError(RuntimeError):
    pass


class GridDesc(C.Structure):
    _fields_ = [("kind", C.c_int), ("r_max", C.c_double), ("z_min", C.c_double), ("z_max", C.c_double),
                ("nr", C.c_int), ("nz", C.c_int), ("levels", C.c_int)]


class SpeciesDesc(C.Structure):
    _fields_ = [("mass", C.c_double), ("charge", C.c_double), ("grid", C.c_int)]


class QuadratureDesc(C.Structure):
    _fields_ = [("degree", C.c_int), ("n_gauss_1d", C.c_int)]


_lib = None


def load():
    """Load liblandau_b200.so (built by paper_2209_03228_b200/build.py).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise LandauError("CUDA library %s is missing: run `python -c 'import __graft_entry__ as g; g.build()'`; "
                              "there is no CPU fallback" % LIB_PATH)
        lib = C.CDLL(LIB_PATH)
        lib.landau_last_error.restype = C.c_char_p
        lib.landau_last_error.argtypes = [C.c_void_p]
        lib.landau_launch_count.restype = C.c_longlong
        lib.landau_launch_count.argtypes = [C.c_void_p]
        lib.landau_destroy.restype = None
        lib.landau_destroy.argtypes = [C.c_void_p]
        _lib = lib
    return _lib


def _check(rc, ctx=None):
    if rc != LANDAU_OK:
        msg = load().landau_last_error(ctx)
        raise LandauError("%s: %s" % (STATUS.get(rc, rc), msg.decode() if msg else ""))


def landau_last_error(ctx=None):
    msg = load().landau_last_error(ctx)
    return msg.decode() if msg else ""


def _np(a):
    return a.ctypes.data_as(C.c_void_p)


def _stream(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    return C.c_void_p(int(stream))


def _dev_ptr(t):
    import torch
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def landau_create(grids, species, quadrature, nu=None, cuda_device=0):
    """grids: list of dict(kind,r_max,z_min,z_max,nr,nz,levels); species: list of dict(mass,charge,grid);
    quadrature: dict(degree, n_gauss_1d) or an int degree.  Returns an opaque context handle (c_void_p)."""
    lib = load()
    if isinstance(quadrature, int):
        quadrature = dict(degree=quadrature, n_gauss_1d=quadrature + 1)
    g_arr = (GridDesc * len(grids))(*[GridDesc(int(g["kind"]), float(g["r_max"]), float(g["z_min"]), float(g["z_max"]),
                                               int(g["nr"]), int(g["nz"]), int(g.get("levels", 0))) for g in grids])
    s_arr = (SpeciesDesc * len(species))(*[SpeciesDesc(float(s["mass"]), float(s["charge"]), int(s["grid"]))
                                           for s in species])
    qd = QuadratureDesc(int(quadrature["degree"]), int(quadrature["n_gauss_1d"]))
    nu_arr = None if nu is None else np.ascontiguousarray(nu, dtype=np.float64)
    ctx = C.c_void_p()
    rc = lib.landau_create(g_arr, C.c_int(len(grids)), s_arr, C.c_int(len(species)), C.byref(qd),
                           None if nu_arr is None else _np(nu_arr), C.c_int(cuda_device), C.byref(ctx))
    _check(rc, None)
    return ctx


class MeshDesc(C.Structure):
    _fields_ = [("n_vertices", C.c_int), ("vertices_rz", C.c_void_p), ("n_cells", C.c_int), ("cells", C.c_void_p),
                ("vertices_per_cell", C.c_int)]


def landau_create_meshes(meshes, species, quadrature, nu=None, cuda_device=0):
    """meshes: list of (vertices [nv, 2] (r, z), cells [nc, 4] (quadrilaterals) or [nc, 3] (triangles), counter-clockwise
    vertex ids); otherwise as landau_create."""
    lib = load()
    if isinstance(quadrature, int):
        quadrature = dict(degree=quadrature, n_gauss_1d=quadrature + 1)
    vs = [np.ascontiguousarray(m[0], dtype=np.float64) for m in meshes]
    cs = [np.ascontiguousarray(m[1], dtype=np.int32) for m in meshes]
    m_arr = (MeshDesc * len(meshes))(*[MeshDesc(len(v), v.ctypes.data, len(c), c.ctypes.data, int(c.shape[1]))
                                       for v, c in zip(vs, cs)])
    s_arr = (SpeciesDesc * len(species))(*[SpeciesDesc(float(s["mass"]), float(s["charge"]), int(s["grid"]))
                                           for s in species])
    qd = QuadratureDesc(int(quadrature["degree"]), int(quadrature["n_gauss_1d"]))
    nu_arr = None if nu is None else np.ascontiguousarray(nu, dtype=np.float64)
    ctx = C.c_void_p()
    rc = lib.landau_create_meshes(m_arr, C.c_int(len(meshes)), s_arr, C.c_int(len(species)), C.byref(qd),
                                  None if nu_arr is None else _np(nu_arr), C.c_int(cuda_device), C.byref(ctx))
    _check(rc, None)
    return ctx


def landau_destroy(ctx):
    load().landau_destroy(ctx)


def landau_sizes(ctx, n_grids):
    n_dof, nnz, n_ip, n_cells = (np.zeros(n_grids, np.int32) for _ in range(4))
    fs, vs = C.c_longlong(), C.c_longlong()
    _check(load().landau_sizes(ctx, _np(n_dof), _np(nnz), _np(n_ip), _np(n_cells), C.byref(fs), C.byref(vs)), ctx)
    return dict(n_dof=n_dof, nnz=nnz, n_ip=n_ip, n_cells=n_cells, f_stride=fs.value, csr_stride=vs.value)


def landau_dof_coords(ctx, grid, n_dof):
    rz = np.zeros((n_dof, 2))
    _check(load().landau_dof_coords(ctx, C.c_int(grid), _np(rz)), ctx)
    return rz


def landau_ip_table(ctx, grid, n_ip):
    r, z, w = np.zeros(n_ip), np.zeros(n_ip), np.zeros(n_ip)
    _check(load().landau_ip_table(ctx, C.c_int(grid), _np(r), _np(z), _np(w)), ctx)
    return r, z, w


def landau_csr_pattern(ctx, grid):
    """Device pointers (ints) of rowptr / colidx, owned by the context."""
    rp, ci = C.c_void_p(), C.c_void_p()
    _check(load().landau_csr_pattern(ctx, C.c_int(grid), C.byref(rp), C.byref(ci)), ctx)
    return rp.value, ci.value


def landau_csr_pattern_host(ctx, grid, n_dof, nnz):
    rp, ci = np.zeros(n_dof + 1, np.int32), np.zeros(nnz, np.int32)
    _check(load().landau_csr_pattern_host(ctx, C.c_int(grid), _np(rp), _np(ci)), ctx)
    return rp, ci


def landau_jacobian(ctx, batch_f, batch, dt, out_csr_vals, stream=None):
    """batch_f / out_csr_vals: CUDA float64 torch tensors (device path).  Asynchronous on `stream`."""
    _check(load().landau_jacobian(ctx, _dev_ptr(batch_f), C.c_int(batch), C.c_double(dt), _dev_ptr(out_csr_vals),
                                  _stream(stream)), ctx)


def landau_apply(ctx, batch_f, batch, out_rhs, stream=None):
    _check(load().landau_apply(ctx, _dev_ptr(batch_f), C.c_int(batch), _dev_ptr(out_rhs), _stream(stream)), ctx)


def landau_spmv(ctx, csr_vals, x, batch, y, stream=None):
    _check(load().landau_spmv(ctx, _dev_ptr(csr_vals), _dev_ptr(x), C.c_int(batch), _dev_ptr(y), _stream(stream)), ctx)


def landau_solve(ctx, csr_vals, rhs, batch, rtol, max_it, x, iters=None, relres=None, stream=None):
    """x: initial guess in, solution out.  iters (int32 CUDA tensor [batch, S]) / relres (float64) optional."""
    ip = C.c_void_p(iters.data_ptr()) if iters is not None else None
    rp = C.c_void_p(relres.data_ptr()) if relres is not None else None
    _check(load().landau_solve(ctx, _dev_ptr(csr_vals), _dev_ptr(rhs), C.c_int(batch), C.c_double(rtol), C.c_int(max_it),
                               _dev_ptr(x), ip, rp, _stream(stream)), ctx)


def landau_solve_noalloc(ctx, csr_vals, rhs, batch, rtol, max_it, x, iters=None, relres=None, stream=None):
    """landau_solve for callers whose application owns the device memory (or whose loop cannot take cudaMalloc's
    synchronisation): the Krylov workspace of large systems is a fixed 32 MiB array inside the library, nothing is
    allocated.  Same arguments and results as landau_solve; raises LandauError when the batch needs more than the array
    holds.  One array per device: do not let two calls overlap on the GPU."""
    ip = C.c_void_p(iters.data_ptr()) if iters is not None else None
    rp = C.c_void_p(relres.data_ptr()) if relres is not None else None
    _check(load().landau_solve_noalloc(ctx, _dev_ptr(csr_vals), _dev_ptr(rhs), C.c_int(batch), C.c_double(rtol),
                                       C.c_int(max_it), _dev_ptr(x), ip, rp, _stream(stream)), ctx)


def landau_jacobian_apply(ctx, batch_f, batch, dt, out_csr_vals, out_rhs, stream=None):
    _check(load().landau_jacobian_apply(ctx, _dev_ptr(batch_f), C.c_int(batch), C.c_double(dt), _dev_ptr(out_csr_vals),
                                        _dev_ptr(out_rhs), _stream(stream)), ctx)


def landau_step(ctx, u, batch, dt, newton_rtol, max_newton, lin_rtol, lin_max_it, stream=None):
    """u: u^k in, u^{k+1} out.  Returns dict(newton_its, last_update, lin_half_steps_max, lin_failed, converged);
    LANDAU_NOT_CONVERGED is reported through converged = False (u then holds the last iterate), every other failure raises."""
    info = (C.c_double * 4)()
    rc = load().landau_step(ctx, _dev_ptr(u), C.c_int(batch), C.c_double(dt), C.c_double(newton_rtol), C.c_int(max_newton),
                            C.c_double(lin_rtol), C.c_int(lin_max_it), info, _stream(stream))
    if rc != LANDAU_NOT_CONVERGED:
        _check(rc, ctx)
    return dict(newton_its=int(info[0]), last_update=float(info[1]), lin_half_steps_max=int(info[2]),
                lin_failed=int(info[3]), converged=rc == LANDAU_OK)


def _host_ptr(a):
    """numpy array or CPU (pinned) torch tensor -> pointer."""
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags.c_contiguous
        return _np(a)
    assert not a.is_cuda and a.is_contiguous()
    return C.c_void_p(a.data_ptr())


def landau_jacobian_host(ctx, batch_f_host, batch, dt, out_csr_vals_host, stream=None):
    """HOST buffers in and out (numpy or pinned torch tensors); H2D/D2H copies inside the call; synchronous."""
    _check(load().landau_jacobian_host(ctx, _host_ptr(batch_f_host), C.c_int(batch), C.c_double(dt),
                                       _host_ptr(out_csr_vals_host), _stream(stream)), ctx)


def landau_apply_host(ctx, batch_f_host, batch, out_rhs_host, stream=None):
    _check(load().landau_apply_host(ctx, _host_ptr(batch_f_host), C.c_int(batch), _host_ptr(out_rhs_host),
                                    _stream(stream)), ctx)


def landau_last_coefficients(ctx, n_entries, dk_stride):
    """Coefficients of the first `n_entries` entries of the last pass: array [n_entries * dk_stride]."""
    out = np.zeros(int(n_entries) * int(dk_stride))
    _check(load().landau_last_coefficients(ctx, _np(out), C.c_int(n_entries)), ctx)
    return out


def landau_reserve(ctx, max_batch):
    _check(load().landau_reserve(ctx, C.c_int(max_batch)), ctx)


def landau_tensor_eval(r, z, rb, zb, out, stream=None):
    _check(load().landau_tensor_eval(_dev_ptr(r), _dev_ptr(z), _dev_ptr(rb), _dev_ptr(zb), C.c_int(r.numel()),
                                     _dev_ptr(out), _stream(stream)))


def landau_ellip_eval(m, mp, out, stream=None):
    _check(load().landau_ellip_eval(_dev_ptr(m), _dev_ptr(mp), C.c_int(m.numel()), _dev_ptr(out), _stream(stream)))


def landau_fp64_probe(kind, iters=20000, stream=None):
    t = C.c_double()
    _check(load().landau_fp64_probe(C.c_int(kind), C.c_int(iters), C.byref(t), _stream(stream)))
    return t.value


def landau_l2_probe(nbytes=32 << 20, iters=64, stream=None):
    """L2 -> SM read bandwidth in GB/s on a buffer of nbytes that stays L2-resident."""
    t = C.c_double()
    _check(load().landau_l2_probe(C.c_longlong(nbytes), C.c_int(iters), C.byref(t), _stream(stream)))
    return t.value


def landau_launch_count(ctx):
    return int(load().landau_launch_count(ctx))


def landau_is_separable(ctx):
    rc = load().landau_is_separable(ctx)
    if rc < 0:
        _check(rc, ctx)
    return bool(rc)


def landau_set_timing(ctx, enabled):
    _check(load().landau_set_timing(ctx, C.c_int(1 if enabled else 0)), ctx)


def landau_last_stage_ms(ctx):
    ms = (C.c_float * 4)()
    _check(load().landau_last_stage_ms(ctx, ms), ctx)
    return [float(x) for x in ms]


def landau_set_inner_kernel(ctx, which):
    _check(load().landau_set_inner_kernel(ctx, C.c_int(which)), ctx)


def landau_set_assembly_kernel(ctx, which):
    _check(load().landau_set_assembly_kernel(ctx, C.c_int(which)), ctx)


def landau_solve_matrix_in_shared(ctx):
    """True when the solve copies every system's matrix to shared memory once (small systems); False: streamed from L2."""
    m = C.c_int(-1)
    _check(load().landau_solve_mode(ctx, None, None, C.byref(m)), ctx)
    return bool(m.value)


def landau_set_solve_kernel(ctx, which):
    _check(load().landau_set_solve_kernel(ctx, C.c_int(which)), ctx)


def landau_solve_mode(ctx):
    """(warps per block of the warp-per-system kernel, or 0 when one thread block per system runs; largest n_dof)."""
    w, n, m = C.c_int(-1), C.c_int(-1), C.c_int(-1)
    _check(load().landau_solve_mode(ctx, C.byref(w), C.byref(n), C.byref(m)), ctx)
    return w.value, n.value


def landau_assembly_info(ctx, grid):
    rc, ns, nsimple = C.c_int(), C.c_int(), C.c_int()
    _check(load().landau_assembly_info(ctx, C.c_int(grid), C.byref(rc), C.byref(ns), C.byref(nsimple)), ctx)
    return dict(ring_cells=rc.value, n_steps=ns.value, n_simple_slots=nsimple.value)


def landau_set_batch_chunk(ctx, chunk):
    _check(load().landau_set_batch_chunk(ctx, C.c_int(chunk)), ctx)


class Landau:
    """Convenience owner of one context (still marshalling only)."""

    def __init__(self, grids, species, degree, nu=None, device=0):
        self.G, self.S = len(grids), len(species)
        self.species = [dict(s) for s in species]
        self.sgrid = [int(s["grid"]) for s in species]
        self.ctx = landau_create(grids, species, degree, nu, device)
        self._sizes()

    @classmethod
    def from_meshes(cls, meshes, species, degree, nu=None, device=0):
        """Unstructured quadrilateral grids (landau_create_meshes)."""
        self = cls.__new__(cls)
        self.G, self.S, self.degree = len(meshes), len(species), degree
        self.sgrid = [int(s["grid"]) for s in species]
        self.ctx = landau_create_meshes(meshes, species, degree, nu, device)
        self._sizes()
        return self

    def _sizes(self):
        sz = landau_sizes(self.ctx, self.G)
        self.n_dof, self.nnz, self.n_ip, self.n_cells = sz["n_dof"], sz["nnz"], sz["n_ip"], sz["n_cells"]
        self.f_stride, self.csr_stride = sz["f_stride"], sz["csr_stride"]
        self.f_off = np.concatenate([[0], np.cumsum([self.n_dof[g] for g in self.sgrid])]).astype(np.int64)
        self.v_off = np.concatenate([[0], np.cumsum([self.nnz[g] for g in self.sgrid])]).astype(np.int64)
        self.dk_stride = int(sum(5 * self.n_ip[g] for g in self.sgrid))

    def close(self):
        if self.ctx is not None:
            landau_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def dof_coords(self, g):
        return landau_dof_coords(self.ctx, g, int(self.n_dof[g]))

    def ip_table(self, g):
        return landau_ip_table(self.ctx, g, int(self.n_ip[g]))

    def pattern(self, g):
        return landau_csr_pattern_host(self.ctx, g, int(self.n_dof[g]), int(self.nnz[g]))

    def jacobian(self, batch_f, dt, out=None, stream=None):
        import torch
        B = batch_f.shape[0]
        if out is None:
            out = torch.empty((B, self.csr_stride), dtype=torch.float64, device=batch_f.device)
        landau_jacobian(self.ctx, batch_f, B, dt, out, stream)
        return out

    def apply(self, batch_f, out=None, stream=None):
        import torch
        B = batch_f.shape[0]
        if out is None:
            out = torch.empty((B, self.f_stride), dtype=torch.float64, device=batch_f.device)
        landau_apply(self.ctx, batch_f, B, out, stream)
        return out

    def spmv(self, csr_vals, x, stream=None):
        import torch
        y = torch.empty_like(x)
        landau_spmv(self.ctx, csr_vals, x, x.shape[0], y, stream)
        return y

    def solve(self, csr_vals, rhs, rtol=1e-10, max_it=200, x0=None, stream=None):
        """Returns (x, half-steps [B, S] int32, residual bounds [B, S])."""
        import torch
        B = rhs.shape[0]
        x = torch.zeros_like(rhs) if x0 is None else x0.clone()
        iters = torch.zeros((B, self.S), dtype=torch.int32, device=rhs.device)
        relres = torch.zeros((B, self.S), dtype=torch.float64, device=rhs.device)
        landau_solve(self.ctx, csr_vals, rhs, B, rtol, max_it, x, iters, relres, stream)
        return x, iters, relres

    def solve_noalloc(self, csr_vals, rhs, x, iters, relres, rtol=1e-10, max_it=200, stream=None):
        """landau_solve_noalloc on buffers the CALLER owns (nothing is allocated here either): x holds the initial guess on
        entry and the solution on return; iters [B, S] int32 and relres [B, S] float64 may be None."""
        landau_solve_noalloc(self.ctx, csr_vals, rhs, rhs.shape[0], rtol, max_it, x, iters, relres, stream)

    def step(self, u, dt, newton_rtol=1e-10, max_newton=50, lin_rtol=1e-12, lin_max_it=1000, stream=None):
        """Backward-Euler step in place (u: [B, f_stride] CUDA float64)."""
        return landau_step(self.ctx, u, u.shape[0], dt, newton_rtol, max_newton, lin_rtol, lin_max_it, stream)

    def last_coefficients(self, batch):
        """list over species of arrays [batch, 5, n_ip]."""
        raw = landau_last_coefficients(self.ctx, batch, self.dk_stride).reshape(batch, self.dk_stride)
        out, o = [], 0
        for g in self.sgrid:
            n = 5 * int(self.n_ip[g])
            out.append(raw[:, o:o + n].reshape(batch, 5, -1))
            o += n
        return out
