"""GPU test of landau_solve_noalloc, the batched solve for callers that cannot let the library allocate device memory
(an application whose own pool already owns the card, or a time-step loop that cannot take the device-wide
synchronisation of cudaMalloc / cudaFree).  landau_solve keeps the Krylov vectors of systems too large for shared memory
in a workspace it grows with cudaMalloc; landau_solve_noalloc runs the same kernel with those vectors in a fixed 32 MiB
array that is part of the library image.

What is checked: on a context that really uses the workspace (electrons on a uniform 16 x 32 Q3 grid, 4,753 unknowns,
more than the ~4,100 whose vectors fit in an SM's shared memory; deuterium on a small grid whose vectors do fit, so one
launch mixes both kinds of system), two calls IN A ROW with different right-hand sides each reproduce landau_solve to the
1e-10 relative bar per (entry, species) block that the parity tests of this repository use -- the second call finds the
first call's vectors in the array and must not be disturbed by them.  Both solutions are also checked against the
systems themselves (true residual through landau_spmv), and a batch that needs more than the array holds must be refused
with a message that says so.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It does not depend on anything the other tests leave behind (run it alone: `pytest tests/test_zz_no_alloc.py -m gpu`)."""
import math

import numpy as np
import pytest

from paper_2209_03228_b200 import workloads as W

pytestmark = pytest.mark.gpu

RTOL_PARITY = 1e-10   # the per-block bar of the parity tests (north_star)
WS_BYTES = 32 << 20   # LANDAU_SOLVE_NOALLOC_WS_BYTES of include/landau.h


def _large_system_config(batch):
    """Config 5's recipe (e- / D+, Q3, shifted Maxwellians) with the electron grid grown to 16 x 32 cells."""
    md = 3670.0
    grids = [W._grid(0, 5.0, 16, 32), W._grid(0, 5.0 / math.sqrt(md), 4, 8)]
    return dict(name="noalloc_eD_16x32_Q3", index=5, grids=grids,
                species=[dict(mass=1.0, charge=-1.0, grid=0), dict(mass=md, charge=1.0, grid=1)],
                degree=3, dt=1.0, batch=batch, state="shifted", alpha=[1.0, 1.0])


def _block_errors(L, a, b):
    """Largest relative difference over the (entry, species) blocks of two [B, f_stride] arrays."""
    worst = 0.0
    for e in range(a.shape[0]):
        for s in range(L.S):
            sl = slice(L.f_off[s], L.f_off[s + 1])
            worst = max(worst, float(np.linalg.norm(a[e, sl] - b[e, sl]) / np.linalg.norm(b[e, sl])))
    return worst


def test_noalloc_solve_matches_landau_solve_on_two_calls_in_a_row():
    import torch
    from paper_2209_03228_b200 import binding as Bn
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    Bn.load()
    B = 5
    cfg = _large_system_config(B)
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    n_e = int(L.f_off[1] - L.f_off[0])
    assert n_e == 4753 and 7 * n_e * 8 > 227 * 1024, "the electron block must be too large for shared memory"
    f = torch.tensor(W.make_batch_f(cfg, [L.dof_coords(g) for g in range(L.G)], batch=B), device="cuda")
    dt = cfg["dt"]
    a_dt = L.jacobian(f, dt)
    rhs1 = L.spmv(a_dt - L.jacobian(f, float("inf")), f)                       # (M/dt) f: the implicit step's own system
    rng = np.random.default_rng(20260311)
    rhs2 = torch.tensor(rng.standard_normal(tuple(rhs1.shape)), device="cuda") * rhs1.abs().mean()
    rtol, max_it = 1e-10, 4000

    # the existing path (workspace from cudaMalloc)
    ref1, it_ref1, _ = L.solve(a_dt, rhs1, rtol=rtol, max_it=max_it)
    ref2, it_ref2, _ = L.solve(a_dt, rhs2, rtol=rtol, max_it=max_it)
    assert int(it_ref1.min()) > 0 and int(it_ref2.min()) > 0, "reference solves must converge"

    # the entry point under test, two calls in a row on caller-owned buffers; the second starts from the array as the
    # first left it
    x1, x2 = torch.zeros_like(rhs1), torch.zeros_like(rhs2)
    it1 = torch.zeros((B, L.S), dtype=torch.int32, device="cuda")
    it2 = torch.zeros_like(it1)
    rr1 = torch.zeros((B, L.S), dtype=torch.float64, device="cuda")
    rr2 = torch.zeros_like(rr1)
    L.solve_noalloc(a_dt, rhs1, x1, it1, rr1, rtol=rtol, max_it=max_it)
    L.solve_noalloc(a_dt, rhs2, x2, it2, rr2, rtol=rtol, max_it=max_it)
    torch.cuda.synchronize()

    assert _block_errors(L, x1.cpu().numpy(), ref1.cpu().numpy()) <= RTOL_PARITY
    assert _block_errors(L, x2.cpu().numpy(), ref2.cpu().numpy()) <= RTOL_PARITY
    assert torch.equal(it1, it_ref1) and torch.equal(it2, it_ref2)            # same iteration, step for step
    assert float(rr1.max()) <= rtol and float(rr2.max()) <= rtol

    # both are solutions of the systems themselves, not just equal to each other
    for x, rhs in ((x1, rhs1), (x2, rhs2)):
        res = (rhs - L.spmv(a_dt, x)).cpu().numpy()
        assert _block_errors(L, res + rhs.cpu().numpy(), rhs.cpu().numpy()) <= 1e-7

    # a third call with a shorter batch (part of the array keeps stale vectors of the longer calls)
    x3 = torch.zeros_like(rhs1[:2])
    L.solve_noalloc(a_dt[:2].contiguous(), rhs1[:2].contiguous(), x3, None, None, rtol=rtol, max_it=max_it)
    assert _block_errors(L, x3.cpu().numpy(), ref1[:2].cpu().numpy()) <= RTOL_PARITY

    # beyond the array: 7 vectors x 4,753 unknowns x 2 species x 8 bytes per entry -> 63 entries fit, 64 do not
    per_entry = 7 * n_e * L.S * 8
    too_many = WS_BYTES // per_entry + 1
    assert too_many == 64
    big_vals = torch.zeros((too_many, a_dt.shape[1]), dtype=torch.float64, device="cuda")
    big_rhs = torch.zeros((too_many, rhs1.shape[1]), dtype=torch.float64, device="cuda")
    big_x = torch.zeros_like(big_rhs)
    with pytest.raises(Bn.LandauError) as err:
        L.solve_noalloc(big_vals, big_rhs, big_x, None, None, rtol=rtol, max_it=10)
    assert "LANDAU_SOLVE_NOALLOC_WS_BYTES" in str(err.value) and "batch = 63" in str(err.value)
    # the refusal leaves the context usable
    x4 = torch.zeros_like(rhs2)
    L.solve_noalloc(a_dt, rhs2, x4, None, None, rtol=rtol, max_it=max_it)
    assert _block_errors(L, x4.cpu().numpy(), ref2.cpu().numpy()) <= RTOL_PARITY
    L.close()


def test_noalloc_solve_on_systems_that_need_no_workspace():
    """Contexts whose systems all fit in shared memory never touch the array and have no batch limit: same results as
    landau_solve on a small quadtree problem."""
    import torch
    from paper_2209_03228_b200 import binding as Bn
    Bn.load()
    B = 7
    cfg = W.tiny_config("quadtree", 3, batch=B)
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    f = torch.tensor(W.make_batch_f(cfg, [L.dof_coords(g) for g in range(L.G)], batch=B), device="cuda")
    a_dt = L.jacobian(f, cfg["dt"])
    rhs = L.spmv(a_dt - L.jacobian(f, float("inf")), f)
    ref, it_ref, _ = L.solve(a_dt, rhs, rtol=1e-12, max_it=400)
    for _ in range(2):
        x = torch.zeros_like(rhs)
        it = torch.zeros((B, L.S), dtype=torch.int32, device="cuda")
        L.solve_noalloc(a_dt, rhs, x, it, None, rtol=1e-12, max_it=400)
        assert _block_errors(L, x.cpu().numpy(), ref.cpu().numpy()) <= RTOL_PARITY
        assert torch.equal(it, it_ref)
    L.close()
