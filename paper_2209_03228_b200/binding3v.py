"""Thin ctypes binding of include/landau3v.h (argument marshalling only -- every step runs in the CUDA kernels).

Same library (liblandau_b200.so), same conventions as binding.py: functions carry the C names, PyTorch is used by callers
for device memory and streams only, there is no CPU fallback (load() raises if the library is missing).
"""
import ctypes as C

import numpy as np

from . import binding as _b

LandauError = _b.LandauError

# every symbol include/landau3v.h declares (tests check the header, this list and the library's exports against each other)
SYMBOLS = ["landau3v_create", "landau3v_destroy", "landau3v_sizes", "landau3v_dof_coords", "landau3v_ip_table",
           "landau3v_csr_pattern", "landau3v_csr_pattern_host", "landau3v_jacobian", "landau3v_apply",
           "landau3v_jacobian_host", "landau3v_jacobian_apply", "landau3v_spmv", "landau3v_solve", "landau3v_step",
           "landau3v_last_coefficients", "landau3v_set_timing", "landau3v_last_stage_ms",
           "landau3v_launch_count", "landau3v_set_inner_kernel", "landau3v_set_assembly_kernel", "landau3v_set_batch_chunk",
           "landau3v_last_error"]


class GridDesc3(C.Structure):
    _fields_ = [("half_width", C.c_double), ("n", C.c_int), ("levels", C.c_int)]


_configured = False


def load():
    global _configured
    lib = _b.load()
    if not _configured:
        lib.landau3v_last_error.restype = C.c_char_p
        lib.landau3v_last_error.argtypes = [C.c_void_p]
        lib.landau3v_launch_count.restype = C.c_longlong
        lib.landau3v_launch_count.argtypes = [C.c_void_p]
        lib.landau3v_destroy.restype = None
        lib.landau3v_destroy.argtypes = [C.c_void_p]
        _configured = True
    return lib


def _check(rc, ctx=None):
    if rc != _b.LANDAU_OK:
        msg = load().landau3v_last_error(ctx)
        raise LandauError("%s: %s" % (_b.STATUS.get(rc, rc), msg.decode() if msg else ""))


def landau3v_create(grids, species, nu=None, cuda_device=0):
    """grids: list of dict(half, n, levels); species: list of dict(mass, charge, grid).  Returns the context handle."""
    lib = load()
    g_arr = (GridDesc3 * len(grids))(*[GridDesc3(float(g["half"]), int(g["n"]), int(g.get("levels", 0))) for g in grids])
    s_arr = (_b.SpeciesDesc * len(species))(*[_b.SpeciesDesc(float(s["mass"]), float(s["charge"]), int(s["grid"]))
                                              for s in species])
    nu_arr = None if nu is None else np.ascontiguousarray(nu, dtype=np.float64)
    ctx = C.c_void_p()
    rc = lib.landau3v_create(g_arr, C.c_int(len(grids)), s_arr, C.c_int(len(species)),
                             None if nu_arr is None else _b._np(nu_arr), C.c_int(cuda_device), C.byref(ctx))
    _check(rc, None)
    return ctx


def landau3v_destroy(ctx):
    load().landau3v_destroy(ctx)


def landau3v_sizes(ctx, n_grids):
    n_dof, nnz, n_ip, n_cells = (np.zeros(n_grids, np.int32) for _ in range(4))
    fs, vs = C.c_longlong(), C.c_longlong()
    _check(load().landau3v_sizes(ctx, _b._np(n_dof), _b._np(nnz), _b._np(n_ip), _b._np(n_cells), C.byref(fs), C.byref(vs)), ctx)
    return dict(n_dof=n_dof, nnz=nnz, n_ip=n_ip, n_cells=n_cells, f_stride=fs.value, csr_stride=vs.value)


def landau3v_dof_coords(ctx, grid, n_dof):
    xyz = np.zeros((n_dof, 3))
    _check(load().landau3v_dof_coords(ctx, C.c_int(grid), _b._np(xyz)), ctx)
    return xyz


def landau3v_ip_table(ctx, grid, n_ip):
    x, y, z, w = (np.zeros(n_ip) for _ in range(4))
    _check(load().landau3v_ip_table(ctx, C.c_int(grid), _b._np(x), _b._np(y), _b._np(z), _b._np(w)), ctx)
    return x, y, z, w


def landau3v_csr_pattern(ctx, grid):
    rp, ci = C.c_void_p(), C.c_void_p()
    _check(load().landau3v_csr_pattern(ctx, C.c_int(grid), C.byref(rp), C.byref(ci)), ctx)
    return rp.value, ci.value


def landau3v_csr_pattern_host(ctx, grid, n_dof, nnz):
    rp, ci = np.zeros(n_dof + 1, np.int32), np.zeros(nnz, np.int32)
    _check(load().landau3v_csr_pattern_host(ctx, C.c_int(grid), _b._np(rp), _b._np(ci)), ctx)
    return rp, ci


def landau3v_jacobian(ctx, batch_f, batch, dt, out, stream=None):
    _check(load().landau3v_jacobian(ctx, _b._dev_ptr(batch_f), C.c_int(batch), C.c_double(dt), _b._dev_ptr(out),
                                    _b._stream(stream)), ctx)


def landau3v_apply(ctx, batch_f, batch, out, stream=None):
    _check(load().landau3v_apply(ctx, _b._dev_ptr(batch_f), C.c_int(batch), _b._dev_ptr(out), _b._stream(stream)), ctx)


def landau3v_jacobian_apply(ctx, batch_f, batch, dt, out_csr_vals, out_rhs, stream=None):
    _check(load().landau3v_jacobian_apply(ctx, _b._dev_ptr(batch_f), C.c_int(batch), C.c_double(dt), _b._dev_ptr(out_csr_vals),
                                          _b._dev_ptr(out_rhs), _b._stream(stream)), ctx)


def landau3v_spmv(ctx, csr_vals, x, batch, y, stream=None):
    _check(load().landau3v_spmv(ctx, _b._dev_ptr(csr_vals), _b._dev_ptr(x), C.c_int(batch), _b._dev_ptr(y), _b._stream(stream)), ctx)


def landau3v_solve(ctx, csr_vals, rhs, batch, rtol, max_it, x, iters=None, relres=None, stream=None):
    """x: initial guess in, solution out.  iters (int32 CUDA tensor [batch, S]) / relres (float64) optional."""
    ip = C.c_void_p(iters.data_ptr()) if iters is not None else None
    rp = C.c_void_p(relres.data_ptr()) if relres is not None else None
    _check(load().landau3v_solve(ctx, _b._dev_ptr(csr_vals), _b._dev_ptr(rhs), C.c_int(batch), C.c_double(rtol), C.c_int(max_it),
                                 _b._dev_ptr(x), ip, rp, _b._stream(stream)), ctx)


def landau3v_step(ctx, u, batch, dt, newton_rtol, max_newton, lin_rtol, lin_max_it, stream=None):
    """u: u^k in, u^{k+1} out.  Returns dict(newton_its, last_update, lin_half_steps_max, lin_failed, converged);
    LANDAU_NOT_CONVERGED is reported through converged = False (u then holds the last iterate), every other failure raises."""
    info = (C.c_double * 4)()
    rc = load().landau3v_step(ctx, _b._dev_ptr(u), C.c_int(batch), C.c_double(dt), C.c_double(newton_rtol), C.c_int(max_newton),
                              C.c_double(lin_rtol), C.c_int(lin_max_it), info, _b._stream(stream))
    if rc != _b.LANDAU_NOT_CONVERGED:
        _check(rc, ctx)
    return dict(newton_its=int(info[0]), last_update=float(info[1]), lin_half_steps_max=int(info[2]),
                lin_failed=int(info[3]), converged=rc == _b.LANDAU_OK)


def landau3v_jacobian_host(ctx, batch_f_host, batch, dt, out_host, stream=None):
    """batch_f_host / out_host: CPU float64 tensors or numpy arrays (pinned memory makes the copies asynchronous)."""
    def ptr(a):
        return C.c_void_p(a.data_ptr()) if hasattr(a, "data_ptr") else _b._np(a)
    _check(load().landau3v_jacobian_host(ctx, ptr(batch_f_host), C.c_int(batch), C.c_double(dt), ptr(out_host),
                                         _b._stream(stream)), ctx)


def landau3v_last_coefficients(ctx, dk_stride, n_entries):
    out = np.zeros(n_entries * dk_stride)
    _check(load().landau3v_last_coefficients(ctx, _b._np(out), C.c_int(n_entries)), ctx)
    return out


def landau3v_set_timing(ctx, enabled):
    _check(load().landau3v_set_timing(ctx, C.c_int(1 if enabled else 0)), ctx)


def landau3v_last_stage_ms(ctx):
    ms = (C.c_float * 4)()
    _check(load().landau3v_last_stage_ms(ctx, ms), ctx)
    return [float(x) for x in ms]


def landau3v_launch_count(ctx):
    return int(load().landau3v_launch_count(ctx))


def landau3v_set_inner_kernel(ctx, which):
    _check(load().landau3v_set_inner_kernel(ctx, C.c_int(which)), ctx)


def landau3v_set_assembly_kernel(ctx, which):
    _check(load().landau3v_set_assembly_kernel(ctx, C.c_int(which)), ctx)


def landau3v_set_batch_chunk(ctx, chunk):
    _check(load().landau3v_set_batch_chunk(ctx, C.c_int(chunk)), ctx)


def landau3v_last_error(ctx=None):
    msg = load().landau3v_last_error(ctx)
    return msg.decode() if msg else ""


class Landau3V:
    """Convenience holder of a 3V context and its sizes (marshalling only)."""

    def __init__(self, grids, species, nu=None, device=0):
        self.G, self.S = len(grids), len(species)
        self.sgrid = [int(s["grid"]) for s in species]
        self.ctx = landau3v_create(grids, species, nu, device)
        sz = landau3v_sizes(self.ctx, self.G)
        self.n_dof, self.nnz, self.n_ip, self.n_cells = sz["n_dof"], sz["nnz"], sz["n_ip"], sz["n_cells"]
        self.f_stride, self.csr_stride = sz["f_stride"], sz["csr_stride"]
        self.f_off = np.concatenate([[0], np.cumsum([self.n_dof[g] for g in self.sgrid])]).astype(np.int64)
        self.v_off = np.concatenate([[0], np.cumsum([self.nnz[g] for g in self.sgrid])]).astype(np.int64)
        self.dk_stride = int(sum(9 * self.n_ip[g] for g in self.sgrid))

    def close(self):
        if self.ctx is not None:
            landau3v_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def dof_coords(self, g):
        return landau3v_dof_coords(self.ctx, g, int(self.n_dof[g]))

    def ip_table(self, g):
        return landau3v_ip_table(self.ctx, g, int(self.n_ip[g]))

    def pattern(self, g):
        return landau3v_csr_pattern_host(self.ctx, g, int(self.n_dof[g]), int(self.nnz[g]))

    def jacobian(self, batch_f, dt, out=None, stream=None):
        import torch
        B = batch_f.shape[0]
        if out is None:
            out = torch.empty((B, self.csr_stride), dtype=torch.float64, device=batch_f.device)
        landau3v_jacobian(self.ctx, batch_f, B, dt, out, stream)
        return out

    def apply(self, batch_f, out=None, stream=None):
        import torch
        B = batch_f.shape[0]
        if out is None:
            out = torch.empty((B, self.f_stride), dtype=torch.float64, device=batch_f.device)
        landau3v_apply(self.ctx, batch_f, B, out, stream)
        return out

    def jacobian_apply(self, batch_f, dt, stream=None):
        import torch
        B = batch_f.shape[0]
        vals = torch.empty((B, self.csr_stride), dtype=torch.float64, device=batch_f.device)
        rhs = torch.empty((B, self.f_stride), dtype=torch.float64, device=batch_f.device)
        landau3v_jacobian_apply(self.ctx, batch_f, B, dt, vals, rhs, stream)
        return vals, rhs

    def spmv(self, csr_vals, x, stream=None):
        import torch
        y = torch.empty_like(x)
        landau3v_spmv(self.ctx, csr_vals, x, x.shape[0], y, stream)
        return y

    def solve(self, csr_vals, rhs, rtol=1e-10, max_it=200, x0=None, stream=None):
        """Returns (x, half-steps [B, S] int32, residual bounds [B, S])."""
        import torch
        B = rhs.shape[0]
        x = torch.zeros_like(rhs) if x0 is None else x0.clone()
        iters = torch.zeros((B, self.S), dtype=torch.int32, device=rhs.device)
        relres = torch.zeros((B, self.S), dtype=torch.float64, device=rhs.device)
        landau3v_solve(self.ctx, csr_vals, rhs, B, rtol, max_it, x, iters, relres, stream)
        return x, iters, relres

    def step(self, u, dt, newton_rtol=1e-10, max_newton=50, lin_rtol=1e-12, lin_max_it=1000, stream=None):
        """Backward-Euler step in place (u: [B, f_stride] CUDA float64)."""
        return landau3v_step(self.ctx, u, u.shape[0], dt, newton_rtol, max_newton, lin_rtol, lin_max_it, stream)

    def last_coefficients(self, batch):
        """list over species of arrays [batch, 9, n_ip]."""
        flat = landau3v_last_coefficients(self.ctx, self.dk_stride, batch).reshape(batch, self.dk_stride)
        out, off = [], 0
        for s in range(self.S):
            n = int(self.n_ip[self.sgrid[s]])
            out.append(flat[:, off:off + 9 * n].reshape(batch, 9, n))
            off += 9 * n
        return out
