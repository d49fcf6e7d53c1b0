"""Pins of the linear-solve oracle (oracle/solve_oracle.py) against what the mathematics and the paper fix -- none of
them re-calls the routine under test: a manufactured solution, the dense product, discrete density conservation of
the implicit step, and the restated TFQMR iteration against the direct solve."""
import numpy as np
import pytest

from oracle import solve_oracle as SO
from paper_2209_03228_b200 import workloads as W


def _random_csr(n, seed):
    """Diagonally dominant non-symmetric band-ish matrix with a random pattern, columns ascending in each row."""
    rng = np.random.default_rng(seed)
    rowptr, colidx, vals = [0], [], []
    for i in range(n):
        cols = sorted(set([i] + [int(c) for c in rng.integers(max(0, i - 7), min(n, i + 8), size=6)]))
        v = rng.normal(size=len(cols))
        v[cols.index(i)] = 4.0 + np.abs(v).sum()
        colidx += cols
        vals += list(v)
        rowptr.append(len(colidx))
    return np.array(rowptr, np.int32), np.array(colidx, np.int32), np.array(vals)


def test_matvec_is_the_dense_product():
    rp, ci, v = _random_csr(57, 1)
    x = np.random.default_rng(2).normal(size=57)
    assert np.allclose(SO.csr_matvec(rp, ci, v, x), SO.csr_to_dense(rp, ci, v) @ x, rtol=0, atol=1e-13)


def test_manufactured_solution():
    rp, ci, v = _random_csr(83, 3)
    xs = np.random.default_rng(4).normal(size=83)
    b = SO.csr_to_dense(rp, ci, v) @ xs
    assert np.linalg.norm(SO.solve_direct(rp, ci, v, b) - xs) < 1e-13 * np.linalg.norm(xs)
    x, m, ok = SO.tfqmr_reference(rp, ci, v, b, 1e-13, 200)
    assert ok and np.linalg.norm(x - xs) < 1e-11 * np.linalg.norm(xs)
    assert SO.residual(rp, ci, v, x, b) < 1e-12
    # an unreachable tolerance is reported, not hidden
    _, m2, ok2 = SO.tfqmr_reference(rp, ci, v, b, 1e-13, 2)
    assert not ok2 and m2 == 4


@pytest.mark.parametrize("kind", ["uniform", "quadtree"])
def test_implicit_step_conserves_density_and_matches_tfqmr(orc, kind):
    """x = (M/dt - J[f])^{-1} (M/dt) f  keeps  1^T M x = 1^T M f  for every species because the columns of J sum to zero
    (conservative weak form; backward Euler of PAPER.md:75-77)."""
    cfg = W.tiny_config(kind, 2, batch=1)
    o = orc.Oracle(cfg["grids"], cfg["species"], cfg["degree"])
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=1)[0]
    dt = 0.7
    vals = o.jacobian(f, dt)
    for s in range(o.S):
        g = o.sgrid[s]
        rp, ci = o.pattern(g)
        a = vals[o.v_off[s]:o.v_off[s + 1]]
        fs = f[o.f_off[s]:o.f_off[s + 1]]
        mass = o.mass(g)
        b = SO.csr_matvec(rp, ci, mass, fs) / dt
        x = SO.solve_direct(rp, ci, a, b)
        one = np.ones_like(fs)
        m_x = one @ SO.csr_matvec(rp, ci, mass, x)
        m_f = one @ SO.csr_matvec(rp, ci, mass, fs)
        assert abs(m_x - m_f) < 1e-12 * abs(m_f)
        assert np.linalg.norm(x - fs) > 1e-6 * np.linalg.norm(fs)        # the step does something
        xt, m, ok = SO.tfqmr_reference(rp, ci, a, b, 1e-12, 500)
        assert ok and np.linalg.norm(xt - x) < 1e-9 * np.linalg.norm(x)
        assert SO.residual(rp, ci, a, xt, b) < 1e-10
