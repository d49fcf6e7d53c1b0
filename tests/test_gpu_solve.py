"""GPU parity of the batched TFQMR solve and the batched CSR product (C ABI: landau_solve, landau_spmv) against
oracle/solve_oracle.py.  Oracle inputs never come from the CUDA path: either both sides build their own system from the
same seeded f (end-to-end case), or the ORACLE's matrix and right-hand side are handed to the CUDA solver (solver-only
case).  Bars: CSR product 1e-13 relative; solve: true residual <= 1000 rtol and <= 1e-9 relative error against the
direct solve at rtol = 1e-12 on the oracle's own system; 1e-8 end to end (both Jacobians agree to 1e-10)."""
import numpy as np
import pytest

from oracle import solve_oracle as SO
from paper_2209_03228_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def Bn():
    from paper_2209_03228_b200 import binding
    binding.load()
    return binding


def _oracle_systems(o, f, dt):
    """Per entry: oracle CSR values of M/dt - J[f], rhs = (M/dt) f, direct solutions."""
    B = f.shape[0]
    vals = np.stack([o.jacobian(f[b], dt) for b in range(B)])
    rhs = np.zeros_like(f)
    sol = np.zeros_like(f)
    for s in range(o.S):
        g = o.sgrid[s]
        rp, ci = o.pattern(g)
        mass = o.mass(g)
        for b in range(B):
            fs = f[b, o.f_off[s]:o.f_off[s + 1]]
            rhs[b, o.f_off[s]:o.f_off[s + 1]] = SO.csr_matvec(rp, ci, mass, fs) / dt
            sol[b, o.f_off[s]:o.f_off[s + 1]] = SO.solve_direct(rp, ci, vals[b, o.v_off[s]:o.v_off[s + 1]],
                                                                rhs[b, o.f_off[s]:o.f_off[s + 1]])
    return vals, rhs, sol


@pytest.mark.parametrize("kind,degree", [("uniform", 2), ("uniform", 3), ("quadtree", 2), ("quadtree", 3)])
@pytest.mark.parametrize("solve_kernel", [0, 2])   # 0: one thread block per system; 2: these small systems take one warp each
def test_solve_and_spmv_against_oracle(orc, Bn, torch_cuda, kind, degree, solve_kernel):
    torch = torch_cuda
    cfg = W.tiny_config(kind, degree, batch=3)
    o = orc.Oracle(cfg["grids"], cfg["species"], cfg["degree"])
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    Bn.landau_set_solve_kernel(L.ctx, solve_kernel)
    wpc, n_max = Bn.landau_solve_mode(L.ctx)          # the kernel this case means to exercise is the one that runs
    assert n_max == max(int(L.n_dof[g]) for g in range(L.G)) and (4 <= wpc <= 8 if solve_kernel == 2 else wpc == 0)
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=3)
    dt = 0.7
    vals, rhs, sol = _oracle_systems(o, f, dt)
    dv, dr, df = (torch.tensor(a, device="cuda") for a in (vals, rhs, f))
    # CSR product with the oracle's values
    y = L.spmv(dv, df).cpu().numpy()
    for b in range(3):
        for s in range(o.S):
            rp, ci = o.pattern(o.sgrid[s])
            ref = SO.csr_matvec(rp, ci, vals[b, o.v_off[s]:o.v_off[s + 1]], f[b, o.f_off[s]:o.f_off[s + 1]])
            assert np.linalg.norm(y[b, o.f_off[s]:o.f_off[s + 1]] - ref) <= 1e-13 * np.linalg.norm(ref)
    # solver only: the oracle's system solved by the CUDA TFQMR
    rtol = 1e-12
    x, iters, relres = L.solve(dv, dr, rtol=rtol, max_it=400)
    x, iters = x.cpu().numpy(), iters.cpu().numpy()
    assert (iters > 0).all() and float(relres.max()) <= rtol
    for b in range(3):
        for s in range(o.S):
            rp, ci = o.pattern(o.sgrid[s])
            a = vals[b, o.v_off[s]:o.v_off[s + 1]]
            sl = slice(o.f_off[s], o.f_off[s + 1])
            # rtol bounds the Jacobi-preconditioned quasi-residual; the plain residual may be larger by the row scaling
            assert SO.residual(rp, ci, a, x[b, sl], rhs[b, sl]) <= 1000 * rtol
            assert np.linalg.norm(x[b, sl] - sol[b, sl]) <= 1e-9 * np.linalg.norm(sol[b, sl])
            # same iteration as the restated algorithm: half-step counts agree up to the drift of rounding errors
            # over ~100 Krylov steps (summation orders differ; a restart may fall on one side only)
            _, m_ref, ok = SO.tfqmr_reference(rp, ci, a, rhs[b, sl], rtol, 400)
            assert ok and m_ref / 2 - 10 <= int(iters[b, s]) <= 2 * m_ref + 10
    # end to end: Jacobian, right-hand side and solve all on the CUDA path
    a_dt = L.jacobian(df, dt)
    a_inf = L.jacobian(df, float("inf"))
    b_gpu = L.spmv(a_dt - a_inf, df)                      # (M/dt) f
    xg, it2, _ = L.solve(a_dt, b_gpu, rtol=rtol, max_it=400)
    xg = xg.cpu().numpy()
    assert (it2.cpu().numpy() > 0).all()
    for b in range(3):
        for s in range(o.S):
            sl = slice(o.f_off[s], o.f_off[s + 1])
            assert np.linalg.norm(xg[b, sl] - sol[b, sl]) <= 1e-8 * np.linalg.norm(sol[b, sl])
    L.close()


def test_solve_systems_too_large_for_shared_memory(orc, Bn, torch_cuda):
    """systems whose seven Krylov vectors do not fit in an SM's shared memory (more than 4,146 unknowns) keep
    them in a global workspace (PAPER.md:117 discusses scaling the batched solver beyond one processing element's fast
    memory).  Electrons on a uniform 16 x 32 Q3 grid (4,753 unknowns) beside deuterium on a small grid whose vectors do fit:
    the ORACLE's matrices and right-hand sides, CUDA TFQMR against the dense direct solve."""
    import math
    torch = torch_cuda
    md = 3670.0
    cfg = dict(W.config(5), name="eD_16x32_Q3", batch=2,
               grids=[W._grid(0, 5.0, 16, 32), W._grid(0, 5.0 / math.sqrt(md), 4, 8)])
    o = orc.Oracle(cfg["grids"], cfg["species"], cfg["degree"])
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    _, n_max = Bn.landau_solve_mode(L.ctx)
    assert n_max == 4753 and 7 * n_max * 8 > 227 * 1024
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=2)
    vals, rhs, sol = _oracle_systems(o, f, cfg["dt"])
    dv, dr = torch.tensor(vals, device="cuda"), torch.tensor(rhs, device="cuda")
    rtol = 1e-13
    x, iters, relres = L.solve(dv, dr, rtol=rtol, max_it=20000)
    x, iters = x.cpu().numpy(), iters.cpu().numpy()
    assert (iters > 0).all() and float(relres.max()) <= rtol
    for b in range(2):
        for s in range(o.S):
            rp, ci = o.pattern(o.sgrid[s])
            sl = slice(o.f_off[s], o.f_off[s + 1])
            assert SO.residual(rp, ci, vals[b, o.v_off[s]:o.v_off[s + 1]], x[b, sl], rhs[b, sl]) <= 1000 * rtol
            err = np.linalg.norm(x[b, sl] - sol[b, sl]) / np.linalg.norm(sol[b, sl])
            assert err <= 1e-9, (b, s, err)
    L.close()


def test_spmv_rows_longer_than_the_register_window(orc, Bn, torch_cuda):
    """k4_spmv holds 48 entries of a row in registers (8 lanes x 6) and finishes longer rows -- the rows that
    couple through hanging nodes -- in a tail loop.  Config 4's quadtree grids have such rows; seeded values on the
    oracle's pattern, landau_spmv against the plain CSR product, every entry of a small batch."""
    torch = torch_cuda
    cfg = W.config(4)
    o = orc.Oracle(cfg["grids"], cfg["species"], cfg["degree"])
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    longest = 0
    for g in range(o.G):
        rp, ci = o.pattern(g)
        rp2, ci2 = L.pattern(g)
        assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)
        longest = max(longest, int(np.diff(rp).max()))
    assert longest > 48, longest
    B = 3
    rng = np.random.default_rng(404)
    vals = rng.standard_normal((B, L.csr_stride))
    xs = rng.standard_normal((B, L.f_stride))
    y = L.spmv(torch.tensor(vals, device="cuda"), torch.tensor(xs, device="cuda")).cpu().numpy()
    for b in range(B):
        for s in range(o.S):
            rp, ci = o.pattern(o.sgrid[s])
            ref = SO.csr_matvec(rp, ci, vals[b, o.v_off[s]:o.v_off[s + 1]], xs[b, o.f_off[s]:o.f_off[s + 1]])
            got = y[b, o.f_off[s]:o.f_off[s + 1]]
            assert np.linalg.norm(got - ref) <= 1e-13 * np.linalg.norm(ref)
            # row by row too: a wrong tail would hide in the norm of 1,000 short rows
            scale = SO.csr_matvec(rp, ci, np.abs(vals[b, o.v_off[s]:o.v_off[s + 1]]), np.abs(xs[b, o.f_off[s]:o.f_off[s + 1]]))
            assert (np.abs(got - ref) <= 1e-14 * scale * np.diff(rp)).all()
    L.close()


@pytest.mark.parametrize("kind", ["uniform", "quadtree"])
def test_warp_mode_with_ragged_entry_groups(Bn, torch_cuda, kind):
    """the warp-per-system kernel with more entries than warps per block and a last block that is only partly
    filled (its idle warps leave after the shared pattern is loaded), on two grids of different size: same iterates as
    one thread block per system, and true residuals at the tolerance."""
    torch = torch_cuda
    cfg = W.tiny_config(kind, 3, batch=2)
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    assert len({int(L.n_dof[g]) for g in range(L.G)}) == 2
    Bn.landau_set_solve_kernel(L.ctx, 2)
    wpc, _ = Bn.landau_solve_mode(L.ctx)
    assert 4 <= wpc <= 8
    B = 2 * wpc + 3                                   # three blocks per species, the last with 3 of wpc warps at work
    f = torch.tensor(W.make_batch_f(cfg, [L.dof_coords(g) for g in range(L.G)], batch=B), device="cuda")
    a_dt = L.jacobian(f, cfg["dt"])
    rhs = L.spmv(a_dt - L.jacobian(f, float("inf")), f)
    xw, itw, rrw = L.solve(a_dt, rhs, rtol=1e-12, max_it=400)
    Bn.landau_set_solve_kernel(L.ctx, 0)
    assert Bn.landau_solve_mode(L.ctx)[0] == 0
    xc, itc, _ = L.solve(a_dt, rhs, rtol=1e-12, max_it=400)
    assert int(itw.min()) > 0 and int(itc.min()) > 0 and float(rrw.max()) <= 1e-12
    res = rhs - L.spmv(a_dt, xw)
    for s in range(L.S):
        sl = slice(int(L.f_off[s]), int(L.f_off[s + 1]))
        assert float(((xw - xc)[:, sl].norm(dim=1) / xc[:, sl].norm(dim=1)).max()) <= 1e-10
        assert float((res[:, sl].norm(dim=1) / rhs[:, sl].norm(dim=1)).max()) <= 1e-9
    # summation orders differ (32 against 128 partial sums): the counts agree up to the drift the oracle comparison allows
    assert bool(((itw >= itc // 2 - 10) & (itw <= 2 * itc + 10)).all())
    L.close()


def test_solve_edge_cases(orc, Bn, torch_cuda):
    torch = torch_cuda
    cfg = W.tiny_config("uniform", 2, batch=2)
    o = orc.Oracle(cfg["grids"], cfg["species"], cfg["degree"])
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=2)
    vals, rhs, sol = _oracle_systems(o, f, 0.5)
    dv, dr = torch.tensor(vals, device="cuda"), torch.tensor(rhs, device="cuda")
    # too few iterations: reported as not converged, x holds the last iterate
    x, iters, relres = L.solve(dv, dr, rtol=1e-13, max_it=2)
    assert (iters.cpu().numpy() == -5).all() and float(relres.min()) > 1e-13
    # zero right-hand side: x = 0 at once
    x, iters, _ = L.solve(dv, torch.zeros_like(dr), rtol=1e-10, max_it=50)
    assert float(x.abs().max()) == 0.0 and (iters.cpu().numpy() == 0).all()
    # the exact solution as initial guess stops within a few half-steps and stays put
    x0 = torch.tensor(sol, device="cuda")
    x, iters, _ = L.solve(dv, dr, rtol=1e-6, max_it=50, x0=x0)
    assert float((x - x0).norm() / x0.norm()) < 1e-10
    # batch == 0 and bad arguments
    Bn.landau_solve(L.ctx, dv, dr, 0, 1e-8, 10, x)
    with pytest.raises(Bn.LandauError):
        Bn.landau_solve(L.ctx, dv, dr, 2, 0.0, 10, x)
    with pytest.raises(Bn.LandauError):
        Bn.landau_solve(L.ctx, dv, dr, 2, 1e-8, 0, x)
    L.close()


@pytest.mark.parametrize("c,B", [(2, 64), (4, 32), (5, 16)])
def test_implicit_step_properties_at_config_size(Bn, torch_cuda, c, B):
    """Properties that hold at any size, on the CUDA path only: true residual of every block and conservation of
    density by the implicit step, 1^T M x = 1^T M f (columns of J sum to zero)."""
    torch = torch_cuda
    cfg = W.config(c)
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    f = torch.tensor(W.make_batch_f(cfg, [L.dof_coords(g) for g in range(L.G)], batch=B), device="cuda")
    dt = cfg["dt"]
    a_dt, a_inf = L.jacobian(f, dt), L.jacobian(f, float("inf"))
    m_dt = a_dt - a_inf
    rhs = L.spmv(m_dt, f)
    x, iters, relres = L.solve(a_dt, rhs, rtol=1e-9, max_it=1000)
    assert int(iters.min()) > 0, int(iters.min())
    res = rhs - L.spmv(a_dt, x)
    mx, mf = L.spmv(m_dt, x), rhs
    for s in range(L.S):
        sl = slice(int(L.f_off[s]), int(L.f_off[s + 1]))
        assert float((res[:, sl].norm(dim=1) / rhs[:, sl].norm(dim=1)).max()) < 1e-7
        assert float(((mx[:, sl].sum(dim=1) - mf[:, sl].sum(dim=1)).abs() / mf[:, sl].sum(dim=1).abs()).max()) < 1e-7
    L.close()
