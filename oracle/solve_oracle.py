"""CPU oracle of the batched linear solve that follows the Jacobian construction.  TEST INFRASTRUCTURE ONLY.

The paper solves, for every (batch entry, species) block, the shifted system of the implicit advance,
    (M/dt - J[f]) x = b                                   (sec. 2.2, 115-117 sec. 3.2, 127 sec. 4.1),
with a batched TFQMR iteration and Jacobi preconditioning.  The RESULT of that solve has a plain definition -- the
solution of the linear system -- so the oracle is that definition written out: `solve_direct` assembles the block
densely from its CSR arrays and calls LAPACK (numpy.linalg.solve), in FP64.  A product solve at relative tolerance
rtol must agree with it to  cond-independent backward error:  ||b - A x|| <= C rtol ||b||  (checked with `residual`).

`tfqmr_reference` restates the iteration itself (Freund's transpose-free QMR as in Saad, "Iterative methods for
sparse linear systems", Alg. 7.8, left Jacobi preconditioning, x0 = 0, stopping test tau sqrt(m+1) <= rtol ||r0||)
step by step with plain numpy vectors; it is pinned against `solve_direct` and is used to compare iteration counts.
The paper does not print the algorithm (it cites PETSc's KSPTFQMR), so this restatement is DESIGN.md reading A18.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it shares no code with
the product package.
"""
import numpy as np


def csr_to_dense(rowptr, colidx, vals):
    n = len(rowptr) - 1
    a = np.zeros((n, n))
    for i in range(n):
        a[i, colidx[rowptr[i]:rowptr[i + 1]]] = vals[rowptr[i]:rowptr[i + 1]]
    return a


def csr_matvec(rowptr, colidx, vals, x):
    """y = A x, row by row (plain definition of the CSR product)."""
    prod = vals * x[colidx]
    return np.add.reduceat(prod, rowptr[:-1])


def solve_direct(rowptr, colidx, vals, rhs):
    """x = A^{-1} b by dense LU (LAPACK dgesv)."""
    return np.linalg.solve(csr_to_dense(rowptr, colidx, vals), rhs)


def residual(rowptr, colidx, vals, x, rhs):
    """||b - A x||_2 / ||b||_2."""
    return np.linalg.norm(rhs - csr_matvec(rowptr, colidx, vals, x)) / np.linalg.norm(rhs)


def tfqmr_reference(rowptr, colidx, vals, rhs, rtol, max_it, run_cap=600):
    """TFQMR on diag(A)^{-1} A x = diag(A)^{-1} b from x0 = 0.  A run that meets the bound  tau sqrt(k) <= rtol ||r0||
    is checked against the true scaled residual and restarted from the current x if that misses the tolerance (the
    tolerance stays relative to the first residual); a run is also restarted after run_cap half-steps.
    Returns (x, half-steps done, converged)."""
    n = len(rhs)
    diag = np.array([vals[rowptr[i]:rowptr[i + 1]][list(colidx[rowptr[i]:rowptr[i + 1]]).index(i)] for i in range(n)])

    def op(u):
        return csr_matvec(rowptr, colidx, vals, u) / diag

    x = np.zeros(n)
    m = 0
    r0norm = None
    while True:
        r = (rhs - csr_matvec(rowptr, colidx, vals, x)) / diag
        tau = np.linalg.norm(r)
        if r0norm is None:
            r0norm = tau
        if tau <= rtol * r0norm:
            return x, m, True
        if m >= 2 * max_it:
            return x, m, False
        w, u, rs = r.copy(), r.copy(), r.copy()
        au = op(u)
        v = au.copy()
        d = np.zeros(n)
        theta = eta = alpha = 0.0
        rho = float(rs @ r)
        bound_met = False
        k = 0
        while not bound_met and m < 2 * max_it and k < run_cap:
            even = k % 2 == 0
            if even:
                sigma = float(rs @ v)
                if sigma == 0.0:
                    return x, m, False
                alpha = rho / sigma
            w = w - alpha * au
            d = u + (theta * theta * eta / alpha) * d
            theta = np.linalg.norm(w) / tau
            c = 1.0 / np.sqrt(1.0 + theta * theta)
            tau = tau * theta * c
            eta = c * c * alpha
            x = x + eta * d
            m += 1
            if tau * np.sqrt(k + 1.0) <= rtol * r0norm:
                bound_met = True
            elif even:
                u = u - alpha * v
                au = op(u)
            else:
                rho_new = float(rs @ w)
                if rho == 0.0:
                    return x, m, False
                beta = rho_new / rho
                rho = rho_new
                u_new = w + beta * u
                au_new = op(u_new)
                v = au_new + beta * (au + beta * v)
                u, au = u_new, au_new
            k += 1
