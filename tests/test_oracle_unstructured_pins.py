"""Pins of the oracle's unstructured-quadrilateral path (oracle/landau_oracle.cpp, orc_create_meshes; SURVEY 8f rank 4,
PAPER.md:225-229 sec. 5.2, Table 13) -- CPU only.

  U1  Table 13's point count (24 Q3 cells -> 384 integration points), sum of the weights = the exact moment INT r dA of the
      polygonal mesh (pins det J and the r factor on non-affine cells), 1^T M 1 the same
  U2  polynomials of degree <= k in the PHYSICAL coordinates are reproduced, value and gradient (pins J^-T per point)
  U3  a mesh of rectangles through the unstructured path == the pinned rectangular path (dofs matched by coordinates)
  U4  conservation of density, z-momentum and energy to round-off on semicircle meshes; 1^T J = 0
  U5  brute force on a small distorted mesh: dense Jacobian from independently evaluated global shape functions
  U6  the isotropisation rate of PAPER.md App. B on the semicircle mesh
"""
import math
import os

import numpy as np
import pytest

import temperature_moments as TM
from paper_2209_03228_b200 import workloads as W


def _poly_moment(p):
    """INT r dA over a polygon with vertices p[:, (r, z)] (Green's theorem)."""
    s = 0.0
    for i in range(len(p)):
        x0, y0 = p[i]
        x1, y1 = p[(i + 1) % len(p)]
        s += (x0 + x1) * (x0 * y1 - x1 * y0)
    return s / 6.0


def test_U1_table13_point_count_and_weights(orc):
    v, c = W.semicircle_mesh(5.0, 2, 2)
    o = orc.Oracle.from_meshes([(v, c)], [dict(mass=1.0, charge=-1.0, grid=0)], 3)
    assert o.n_cells[0] == 24 and o.n_ip[0] == 384                      # PAPER.md:311 (Table 13): 24 Q3 cells, 384 IPs
    r, z, w = o.ip_table(0)
    exact = sum(_poly_moment(v[q]) for q in c)
    assert abs(w.sum() - exact) < 1e-13 * exact and abs(o.mass(0).sum() - exact) < 1e-13 * exact
    assert np.all(w > 0) and np.all(r > 0) and np.all(r * r + z * z < 25.0)
    o2 = orc.Oracle.from_meshes([W.semicircle_mesh(5.0, 3, 2)], [dict(mass=1.0, charge=-1.0, grid=0)], 2)
    assert o2.n_ip[0] == o2.n_cells[0] * 9                              # (k+1)^2 points per cell
    with pytest.raises(RuntimeError):                                    # a clockwise cell is refused
        orc.Oracle.from_meshes([(v, c[:, ::-1].copy())], [dict(mass=1.0, charge=-1.0, grid=0)], 3)


@pytest.mark.parametrize("k", [2, 3, 4])
def test_U2_physical_polynomials_are_reproduced(orc, k):
    o = orc.Oracle.from_meshes([W.semicircle_mesh(3.0, 2, 2)], [dict(mass=1.0, charge=-1.0, grid=0)], k)
    rz = o.dof_coords(0)
    R, Z = rz[:, 0], rz[:, 1]
    r, z, w = o.ip_table(0)
    if k == 2:
        f, ex = 1 + R - 2 * Z + R * Z - 0.5 * Z * Z + 0.3 * R * R, 1 + r - 2 * z + r * z - 0.5 * z * z + 0.3 * r * r
        gr, gz = 1 + z + 0.6 * r, -2 + r - z
    elif k == 3:
        f, ex = R ** 3 - 2 * R * Z * Z + Z ** 3 + R * Z, r ** 3 - 2 * r * z * z + z ** 3 + r * z
        gr, gz = 3 * r * r - 2 * z * z + z, -4 * r * z + 3 * z * z + r
    else:
        f, ex = R ** 4 - 3 * R * R * Z * Z + Z ** 4 + R * Z, r ** 4 - 3 * r * r * z * z + z ** 4 + r * z
        gr, gz = 4 * r ** 3 - 6 * r * z * z + z, -6 * r * r * z + 4 * z ** 3 + r
    a, b, c = o.fields(f, 0)
    scale = np.abs(ex).max()
    assert np.abs(a - ex).max() < 1e-13 * scale
    assert np.abs(b - gr).max() < 1e-12 * scale and np.abs(c - gz).max() < 1e-12 * scale
    a4, _, _ = o.fields(R ** (k + 1), 0)                                  # degree k + 1 is not in the space: the pin can fail
    assert np.abs(a4 - r ** (k + 1)).max() > 1e-6


def _match(a, b):
    """permutation p with a[p] == b (rows matched by coordinates)."""
    p = np.array([int(np.argmin(((a - x) ** 2).sum(1))) for x in b])
    assert np.abs(a[p] - b).max() < 1e-12 and len(set(p)) == len(p)
    return p


def _dense(o, s, vals):
    g = o.sgrid[s]
    rp, ci = o.pattern(g)
    A = np.zeros((o.n_dof[g], o.n_dof[g]))
    v = vals[o.v_off[s]:o.v_off[s + 1]]
    for i in range(o.n_dof[g]):
        A[i, ci[rp[i]:rp[i + 1]]] = v[rp[i]:rp[i + 1]]
    return A


def test_U3_rectangles_through_the_unstructured_path_equal_the_rectangular_path(orc):
    cfg = W.tiny_config("uniform", 3, batch=1)
    o = orc.Oracle(cfg["grids"], cfg["species"], 3)
    meshes = []
    for g in cfg["grids"]:
        nr, nz = g["nr"], g["nz"]
        vr, vz = np.linspace(0, g["r_max"], nr + 1), np.linspace(g["z_min"], g["z_max"], nz + 1)
        v = np.array([(vr[i], vz[j]) for j in range(nz + 1) for i in range(nr + 1)])
        c = np.array([(j * (nr + 1) + i, j * (nr + 1) + i + 1, (j + 1) * (nr + 1) + i + 1, (j + 1) * (nr + 1) + i)
                      for j in range(nz) for i in range(nr)], dtype=np.int32)
        meshes.append((v, c))
    u = orc.Oracle.from_meshes(meshes, cfg["species"], 3)
    assert list(u.n_dof) == list(o.n_dof) and list(u.nnz) == list(o.nnz)
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(2)], batch=1)[0]
    fu = W.make_batch_f(cfg, [u.dof_coords(g) for g in range(2)], batch=1)[0]
    A, Au = o.jacobian(f, cfg["dt"]), u.jacobian(fu, cfg["dt"])
    r, ru = o.apply(f), u.apply(fu)
    for s in range(2):
        g = o.sgrid[s]
        p = _match(u.dof_coords(g), o.dof_coords(g))
        D, Du = _dense(o, s, A), _dense(u, s, Au)[np.ix_(p, p)]
        assert np.abs(D - Du).max() < 1e-13 * np.abs(D).max()
        blk, blku = r[o.f_off[s]:o.f_off[s + 1]], ru[u.f_off[s]:u.f_off[s + 1]][p]
        assert np.abs(blk - blku).max() < 1e-13 * np.abs(blk).max()


def test_U4_conservation_on_semicircle_meshes(orc):
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=4.0, charge=1.0, grid=1), dict(mass=9.0, charge=2.0, grid=1)]
    meshes = [W.semicircle_mesh(5.0, 2, 2), W.semicircle_mesh(2.5, 2, 3, core=0.4)]
    o = orc.Oracle.from_meshes(meshes, species, 3)
    cfg = dict(index=81, species=species, state="shifted", alpha=[1.0] * 3, batch=1)
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(2)], batch=1)[0]
    rhs = o.apply(f)
    mom, scale = np.zeros(2), np.zeros(2)
    for s, sp in enumerate(species):
        rz = o.dof_coords(sp["grid"])
        blk = rhs[o.f_off[s]:o.f_off[s + 1]]
        assert abs(blk.sum()) < 1e-12 * np.abs(blk).sum()
        for k, psi in enumerate([rz[:, 1], (rz ** 2).sum(1)]):
            mom[k] += sp["mass"] * (psi @ blk)
            scale[k] += sp["mass"] * (np.abs(psi) @ np.abs(blk))
    assert np.all(np.abs(mom) < 1e-12 * scale) and np.abs(rhs).max() > 1e-8
    J = o.jacobian(f, float("inf"))
    for s, sp in enumerate(species):
        rp, ci = o.pattern(sp["grid"])
        v = J[o.v_off[s]:o.v_off[s + 1]]
        col = np.zeros(o.n_dof[sp["grid"]])
        np.add.at(col, ci, v)
        assert np.abs(col).max() < 1e-12 * np.abs(v).max()
        y = np.add.reduceat(v * f[o.f_off[s]:o.f_off[s + 1]][ci], rp[:-1])
        assert np.abs(rhs[o.f_off[s]:o.f_off[s + 1]] + y).max() < 1e-12 * np.abs(y).max()


def _lagrange_eq(k, x):
    nodes = -1.0 + 2.0 * np.arange(k + 1) / k
    val, der = np.zeros(k + 1), np.zeros(k + 1)
    for c in range(k + 1):
        others = [d for d in range(k + 1) if d != c]
        val[c] = np.prod([(x - nodes[d]) / (nodes[c] - nodes[d]) for d in others])
        der[c] = sum(np.prod([(x - nodes[d]) / (nodes[c] - nodes[d]) for d in others if d != e]) / (nodes[c] - nodes[e]) for e in others)
    return val, der


def test_U5_brute_force_on_a_distorted_mesh(orc):
    """Four distorted quadrilaterals around an interior vertex (none a parallelogram).  Global shape functions are evaluated
    independently: reference basis at the Gauss points, physical gradients from solving J^T g = grad_ref with numpy, nodes
    identified by rounding coordinates; azimuthal-quadrature tensor; plain pair loop."""
    k, dt = 2, 0.7
    v = np.array([(0.2, -1.0), (1.1, -1.2), (2.3, -0.9), (0.1, 0.1), (1.3, -0.1), (2.1, 0.2), (0.3, 1.1), (1.0, 1.3), (2.4, 1.0)])
    c = np.array([(0, 1, 4, 3), (1, 2, 5, 4), (3, 4, 7, 6), (4, 5, 8, 7)], dtype=np.int32)
    o = orc.Oracle.from_meshes([(v, c)], [dict(mass=1.0, charge=-1.0, grid=0)], k)
    rz = o.dof_coords(0)
    gx, gw = np.polynomial.legendre.leggauss(k + 1)
    n = o.n_dof[0]
    ip, wt, PH, PR, PZ = [], [], [], [], []
    for q4 in c:
        P = v[q4]
        def xmap(xi, eta):
            N = 0.25 * np.array([(1 - xi) * (1 - eta), (1 + xi) * (1 - eta), (1 + xi) * (1 + eta), (1 - xi) * (1 + eta)])
            return N @ P
        ids = []
        for a2 in range(k + 1):
            for a1 in range(k + 1):
                x = xmap(-1 + 2 * a1 / k, -1 + 2 * a2 / k)
                ids.append(int(np.argmin(((rz - x) ** 2).sum(1))))
                assert np.abs(rz[ids[-1]] - x).max() < 1e-12
        for q2 in range(k + 1):
            for q1 in range(k + 1):
                xi, eta = gx[q1], gx[q2]
                dN = 0.25 * np.array([[-(1 - eta), (1 - eta), (1 + eta), -(1 + eta)], [-(1 - xi), -(1 + xi), (1 + xi), (1 - xi)]])
                Jm = (dN @ P).T                       # [[dr/dxi, dr/deta], [dz/dxi, dz/deta]]
                x = xmap(xi, eta)
                v1, d1 = _lagrange_eq(k, xi)
                v2, d2 = _lagrange_eq(k, eta)
                ph, pr, pz = np.zeros(n), np.zeros(n), np.zeros(n)
                for a2 in range(k + 1):
                    for a1 in range(k + 1):
                        g = np.linalg.solve(Jm.T, np.array([d1[a1] * v2[a2], v1[a1] * d2[a2]]))
                        I = ids[a1 + (k + 1) * a2]
                        ph[I], pr[I], pz[I] = v1[a1] * v2[a2], g[0], g[1]
                ip.append(x); wt.append(gw[q1] * gw[q2] * np.linalg.det(Jm) * x[0]); PH.append(ph); PR.append(pr); PZ.append(pz)
    ip, wt, PH, PR, PZ = map(np.array, (ip, wt, PH, PR, PZ))
    assert np.abs(PH.sum(1) - 1).max() < 1e-13
    f = math.pi ** -1.5 * np.exp(-((rz[:, 0] - 0.3) ** 2 + (rz[:, 1] - 0.1) ** 2))
    fj, frj, fzj = PH @ f, PR @ f, PZ @ f
    nq = len(ip)
    D, K = np.zeros((nq, 2, 2)), np.zeros((nq, 2))
    for i in range(nq):
        for j in range(nq):
            if i == j:
                continue
            U = orc.tensor_quadrature(ip[i, 0], ip[i, 1], ip[j, 0], ip[j, 1], 1500)
            D[i] += wt[j] * fj[j] * np.array([[U[0], U[1]], [U[7], U[2]]])
            K[i] += wt[j] * (np.array([[U[3], U[4]], [U[5], U[6]]]) @ np.array([frj[j], fzj[j]]))
    A = np.zeros((n, n))
    for q in range(nq):
        gphi = np.stack([PR[q], PZ[q]], 0)
        A += wt[q] * (np.outer(PH[q], PH[q]) / dt + gphi.T @ D[q] @ gphi - np.outer(gphi.T @ K[q], PH[q]))
    dense = _dense(o, 0, o.jacobian(f, dt))
    assert np.linalg.norm(dense - A) < 1e-11 * np.linalg.norm(A) and np.abs(dense - A).max() < 1e-11 * np.abs(A).max()
    Mq = (PH * wt[:, None]).T @ PH
    ref_rhs = (Mq / dt - A) @ f
    assert np.linalg.norm(o.apply(f) - ref_rhs) < 1e-10 * np.linalg.norm(ref_rhs)


def test_U6_isotropization_rate_on_the_semicircle_mesh(orc):
    g = TM.golden_rates(os.path.join(os.path.dirname(__file__), "golden", "nrl_rates.txt"))
    alpha = 1.3
    o = orc.Oracle.from_meshes([W.semicircle_mesh(5.0, 5, 5)], [dict(mass=1.0, charge=-1.0, grid=0)], 3)
    rz = o.dof_coords(0)
    f = (1.0 / alpha) * math.pi ** -1.5 * np.exp(-(rz[:, 1] ** 2 + rz[:, 0] ** 2 / alpha))
    rhs = o.apply(f)
    rp, ci = o.pattern(0)
    mf = np.add.reduceat(o.mass(0) * f[ci], rp[:-1])
    n, tperp, tpar = TM.temperatures(mf, rz[:, 0], rz[:, 1], 1.0)
    dperp, dpar = TM.temperature_rates(mf, rhs, rz[:, 0], rz[:, 1], 1.0)
    assert abs(n - 1.0) < 2e-3 and abs(tperp / tpar - alpha) < 3e-3
    assert abs(dperp + 0.5 * dpar) < 1e-12 * abs(dperp)
    nu_t = TM.nrl_isotropization_rate(g["c_iso"], n, 1.0, tperp, tpar)
    assert abs(-dperp / (tperp - tpar) - nu_t) < 1e-2 * nu_t


# ------------------------------------------------------------------------------------------------ simplex cells (P2 - P4)
def _tri_oracle(orc, mesh, k, species=None):
    return orc.Oracle.from_meshes([mesh], species or [dict(mass=1.0, charge=-1.0, grid=0)], k)


@pytest.mark.parametrize("k,npts", [(2, 6), (3, 12), (4, 16)])
def test_S1_simplex_rule_point_counts_and_exactness(orc, k, npts):
    """Tables 11-12: 864 IPs / 144 P2 cells, 816 / 68 P3, 384 / 24 P4 = 6, 12, 16 points per cell; the rule
    must integrate degree 2k exactly (mass matrix of Pk) -- monomials over the unit right triangle: a! b! / (a + b + 2)!."""
    gold = {2: (864, 144), 3: (816, 68), 4: (384, 24)}[k]
    assert gold[0] == gold[1] * npts
    v = np.array([(0.5, 0.0), (1.5, 0.0), (0.5, 1.0)])
    o = _tri_oracle(orc, (v, np.array([(0, 1, 2)], dtype=np.int32)), k)
    assert o.n_ip[0] == npts and o.n_dof[0] == (k + 1) * (k + 2) // 2
    r, z, w = o.ip_table(0)
    x, y, wq = r - 0.5, z, w / r
    assert np.all(wq > 0) and np.all(x > 0) and np.all(y > 0) and np.all(x + y < 1)
    worst = 0.0
    for a in range(2 * k + 1):
        for b in range(2 * k + 1 - a):
            exact = math.factorial(a) * math.factorial(b) / math.factorial(a + b + 2)
            worst = max(worst, abs((wq * x ** a * y ** b).sum() - exact) / exact)
    assert worst < 1e-13
    a = 2 * k + 1                                                     # one degree more is not exact: the pin can fail
    assert abs((wq * x ** a).sum() - 1.0 / ((a + 1) * (a + 2))) > 1e-9


@pytest.mark.parametrize("k", [2, 3, 4])
def test_S2_simplex_polynomial_reproduction_and_weights(orc, k):
    mesh = W.semicircle_triangles(3.0, 2, 2)
    o = _tri_oracle(orc, mesh, k)
    r, z, w = o.ip_table(0)
    exact = sum(_poly_moment(mesh[0][t]) for t in mesh[1])
    assert abs(w.sum() - exact) < 1e-13 * exact and abs(o.mass(0).sum() - exact) < 1e-13 * exact
    rz = o.dof_coords(0)
    R, Z = rz[:, 0], rz[:, 1]
    f = 1 + R - 2 * Z + R * Z - 0.5 * Z * Z + 0.3 * R * R
    ex, gr, gz = 1 + r - 2 * z + r * z - 0.5 * z * z + 0.3 * r * r, 1 + z + 0.6 * r, -2 + r - z
    if k >= 3:
        f, ex = f + R ** 3 - R * Z * Z, ex + r ** 3 - r * z * z
        gr, gz = gr + 3 * r * r - z * z, gz - 2 * r * z
    if k == 4:
        f, ex = f + R * R * Z * Z, ex + r * r * z * z
        gr, gz = gr + 2 * r * z * z, gz + 2 * r * r * z
    a, b, c = o.fields(f, 0)
    scale = np.abs(ex).max()
    assert np.abs(a - ex).max() < 1e-13 * scale
    assert np.abs(b - gr).max() < 2e-12 * scale and np.abs(c - gz).max() < 2e-12 * scale
    a5, _, _ = o.fields(R ** (k + 1), 0)
    assert np.abs(a5 - r ** (k + 1)).max() > 1e-6


def test_S4_simplex_conservation(orc):
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=4.0, charge=1.0, grid=1)]
    meshes = [W.semicircle_triangles(5.0, 2, 2), W.semicircle_triangles(2.5, 2, 1, core=0.6)]
    o = orc.Oracle.from_meshes(meshes, species, 3)
    cfg = dict(index=84, species=species, state="shifted", alpha=[1.0, 1.0], batch=1)
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(2)], batch=1)[0]
    rhs = o.apply(f)
    mom, scale = np.zeros(2), np.zeros(2)
    for s, sp in enumerate(species):
        rz = o.dof_coords(sp["grid"])
        blk = rhs[o.f_off[s]:o.f_off[s + 1]]
        assert abs(blk.sum()) < 1e-12 * np.abs(blk).sum()
        for k, psi in enumerate([rz[:, 1], (rz ** 2).sum(1)]):
            mom[k] += sp["mass"] * (psi @ blk)
            scale[k] += sp["mass"] * (np.abs(psi) @ np.abs(blk))
    assert np.all(np.abs(mom) < 1e-12 * scale) and np.abs(rhs).max() > 1e-8
    J = o.jacobian(f, float("inf"))
    for s, sp in enumerate(species):
        rp, ci = o.pattern(sp["grid"])
        v = J[o.v_off[s]:o.v_off[s + 1]]
        col = np.zeros(o.n_dof[sp["grid"]])
        np.add.at(col, ci, v)
        assert np.abs(col).max() < 1e-12 * np.abs(v).max()


def test_S5_simplex_brute_force(orc):
    """Four triangles around an interior vertex, P3.  The global shape functions come from an independent construction: the
    cubic Lagrange basis of each triangle by inverting the monomial Vandermonde matrix of its nodes in PHYSICAL coordinates
    (so no reference map and no J^-T at all), values and gradients at the oracle's own integration points."""
    k, dt = 3, 0.7
    v = np.array([(0.2, -1.0), (2.3, -0.9), (1.2, 0.1), (0.1, 1.2), (2.4, 1.1)])
    c = np.array([(0, 1, 2), (1, 4, 2), (4, 3, 2), (3, 0, 2)], dtype=np.int32)
    o = _tri_oracle(orc, (v, c), k)
    rz = o.dof_coords(0)
    ipr, ipz, wt = o.ip_table(0)
    n, nq = o.n_dof[0], o.n_ip[0] // 4
    expo = [(a, b) for a in range(k + 1) for b in range(k + 1 - a)]
    PH, PR, PZ = np.zeros((4 * nq, n)), np.zeros((4 * nq, n)), np.zeros((4 * nq, n))
    for e, tri in enumerate(c):
        P = v[tri]
        nodes = [P[0] + (P[1] - P[0]) * i / k + (P[2] - P[0]) * j / k for j in range(k + 1) for i in range(k + 1 - j)]
        ids = [int(np.argmin(((rz - x) ** 2).sum(1))) for x in nodes]
        V = np.array([[x[0] ** a * x[1] ** b for (a, b) in expo] for x in nodes])
        C = np.linalg.inv(V)                                          # column m: monomial coefficients of basis function m
        for q in range(nq):
            x, y = ipr[e * nq + q], ipz[e * nq + q]
            mono = np.array([x ** a * y ** b for (a, b) in expo])
            dmx = np.array([a * x ** (a - 1) * y ** b if a else 0.0 for (a, b) in expo])
            dmy = np.array([b * x ** a * y ** (b - 1) if b else 0.0 for (a, b) in expo])
            PH[e * nq + q, ids], PR[e * nq + q, ids], PZ[e * nq + q, ids] = mono @ C, dmx @ C, dmy @ C
    assert np.abs(PH.sum(1) - 1).max() < 1e-11
    f = math.pi ** -1.5 * np.exp(-((rz[:, 0] - 0.3) ** 2 + (rz[:, 1] - 0.1) ** 2))
    fj, frj, fzj = PH @ f, PR @ f, PZ @ f
    N = 4 * nq
    D, K = np.zeros((N, 2, 2)), np.zeros((N, 2))
    for i in range(N):
        for j in range(N):
            if i == j:
                continue
            U = orc.tensor_quadrature(ipr[i], ipz[i], ipr[j], ipz[j], 1500)
            D[i] += wt[j] * fj[j] * np.array([[U[0], U[1]], [U[7], U[2]]])
            K[i] += wt[j] * (np.array([[U[3], U[4]], [U[5], U[6]]]) @ np.array([frj[j], fzj[j]]))
    A = np.zeros((n, n))
    for q in range(N):
        gphi = np.stack([PR[q], PZ[q]], 0)
        A += wt[q] * (np.outer(PH[q], PH[q]) / dt + gphi.T @ D[q] @ gphi - np.outer(gphi.T @ K[q], PH[q]))
    dense = _dense(o, 0, o.jacobian(f, dt))
    assert np.linalg.norm(dense - A) < 1e-10 * np.linalg.norm(A) and np.abs(dense - A).max() < 1e-10 * np.abs(A).max()
    Mq = (PH * wt[:, None]).T @ PH
    assert np.linalg.norm(o.apply(f) - (Mq / dt - A) @ f) < 1e-9 * np.linalg.norm((Mq / dt - A) @ f)


def test_S6_simplex_isotropization_rate(orc):
    g = TM.golden_rates(os.path.join(os.path.dirname(__file__), "golden", "nrl_rates.txt"))
    alpha = 1.3
    o = _tri_oracle(orc, W.semicircle_triangles(5.0, 4, 4), 3)
    rz = o.dof_coords(0)
    f = (1.0 / alpha) * math.pi ** -1.5 * np.exp(-(rz[:, 1] ** 2 + rz[:, 0] ** 2 / alpha))
    rhs = o.apply(f)
    rp, ci = o.pattern(0)
    mf = np.add.reduceat(o.mass(0) * f[ci], rp[:-1])
    n, tperp, tpar = TM.temperatures(mf, rz[:, 0], rz[:, 1], 1.0)
    dperp, dpar = TM.temperature_rates(mf, rhs, rz[:, 0], rz[:, 1], 1.0)
    assert abs(n - 1.0) < 5e-3 and abs(dperp + 0.5 * dpar) < 1e-12 * abs(dperp)
    nu_t = TM.nrl_isotropization_rate(g["c_iso"], n, 1.0, tperp, tpar)
    assert abs(-dperp / (tperp - tpar) - nu_t) < 2e-2 * nu_t
