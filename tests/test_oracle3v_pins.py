"""Pins of the 3V oracle (oracle/landau3v_oracle.cpp) against what the paper and the mathematics fix -- CPU only.

  T3   tensor identities: U = U^T (by construction of the 6 numbers), U u = 0, trace U = 2/|u|, positive semi-definite,
       value at a hand-computed pair
  M3   the paper's 3V mesh: 120 Q2 cells, 1,045 equations, 54.0 non-zeros per row
  R3   mass = volume to round-off and exact reproduction of tri-quadratic polynomials (value and gradient) through hanging
       faces and edges; partition of unity of the constraint rows
  P5   Rosenbluth closed forms of INT U f and INT U . grad f for a Maxwellian at an exterior point (textbook)
  P6   conservation of density, all three momenta and energy to round-off; 1^T J = 0; apply = -J f
  P8   brute force: dense Jacobian from geometrically built global shape functions (hanging nodes by continuity) and a plain
       pair loop, two species on two grids
  P10  isotropisation rate of a bi-Maxwellian at t = 0 against PAPER.md App. B (fixes nu, t0 and the absence of 2 pi / r
       factors in the Cartesian form)
"""
import math
import os

import numpy as np
import pytest

import temperature_moments as TM


@pytest.fixture(scope="module")
def o3():
    from oracle import oracle3v as O3
    O3.build()
    return O3


def _full(u6):
    return np.array([[u6[0], u6[1], u6[2]], [u6[1], u6[3], u6[4]], [u6[2], u6[4], u6[5]]])


# ------------------------------------------------------------------------------------------------ T3
def test_T3_tensor_identities(o3):
    rng = np.random.default_rng(3)
    for _ in range(200):
        v, vb = rng.normal(size=3) * 3, rng.normal(size=3) * 3
        U = _full(o3.tensor(v, vb))
        u = v - vb
        nu = np.linalg.norm(u)
        assert np.abs(U @ u).max() < 1e-14 * 2 / nu * nu              # null space: U (v - vb) = 0
        assert abs(np.trace(U) - 2 / nu) < 1e-14 * 2 / nu
        ev = np.linalg.eigvalsh(U)
        assert ev[0] > -1e-14 / nu and abs(ev[1] - 1 / nu) < 1e-13 / nu and abs(ev[2] - 1 / nu) < 1e-13 / nu
        assert np.allclose(o3.tensor(vb, v), o3.tensor(v, vb), rtol=0, atol=1e-16 / nu)   # even in u
    # hand-computed: u = (1, 2, 2), |u| = 3: U = (9 I - u u^T) / 27
    U = _full(o3.tensor([1.5, 2.0, 2.5], [0.5, 0.0, 0.5]))
    ref = (9 * np.eye(3) - np.outer([1, 2, 2], [1, 2, 2])) / 27.0
    assert np.abs(U - ref).max() < 1e-16
    assert np.all(o3.tensor([1.0, 2.0, 3.0], [1.0, 2.0, 3.0]) == 0)     # coincident points contribute zero (reading A2)


# ------------------------------------------------------------------------------------------------ M3
def test_M3_paper_mesh_statistics(o3):
    gold = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_mesh_stats.txt")):
        if line.strip() and not line.startswith("#"):
            p = line.split()
            gold[p[0]] = [float(x) for x in p[1:]]
    cells, eqs, nnz_row = gold["throughput_3V_Q2"]
    o = o3.Oracle3V([dict(half=5.0, n=4, levels=1)], [dict(mass=1.0, charge=-1.0, grid=0)])
    assert o.n_cells[0] == cells and o.n_dof[0] == eqs
    assert round(o.nnz[0] / o.n_dof[0], 1) == nnz_row
    assert o.n_ip[0] == cells * 27
    # a uniform grid has the Kronecker counts: (2 n + 1)^3 dofs, rows of 27 / 45 / 75 / 125 entries
    o = o3.Oracle3V([dict(half=1.0, n=3, levels=0)], [dict(mass=1.0, charge=-1.0, grid=0)])
    assert o.n_dof[0] == 7 ** 3 and o.nnz[0] == (3 * 9 - 2) ** 3


# ------------------------------------------------------------------------------------------------ R3
@pytest.mark.parametrize("n,levels", [(4, 1), (3, 1), (4, 2), (2, 0)])
def test_R3_mass_volume_and_polynomial_reproduction(o3, n, levels):
    half = 2.5
    o = o3.Oracle3V([dict(half=half, n=n, levels=levels)], [dict(mass=1.0, charge=-1.0, grid=0)])
    assert abs(o.mass(0).sum() - (2 * half) ** 3) < 1e-12 * (2 * half) ** 3
    x, y, z, w = o.ip_table(0)
    assert abs(w.sum() - (2 * half) ** 3) < 1e-12 * (2 * half) ** 3
    xyz = o.dof_coords(0)
    X, Y, Z = xyz[:, 0], xyz[:, 1], xyz[:, 2]
    # any tri-quadratic polynomial is in the space, hanging nodes included: nodal interpolant == polynomial at the IPs
    f = 0.3 + X * X * Y * Z * Z - 0.7 * X * Y * Y * Z + 0.2 * Z * Z * Y * Y * X * X - X
    fld = o.fields(f, 0)
    ex = 0.3 + x * x * y * z * z - 0.7 * x * y * y * z + 0.2 * z * z * y * y * x * x - x
    gx = 2 * x * y * z * z - 0.7 * y * y * z + 0.4 * x * z * z * y * y - 1
    gy = x * x * z * z - 1.4 * x * y * z + 0.4 * y * z * z * x * x
    gz = 2 * x * x * y * z - 0.7 * x * y * y + 0.4 * z * y * y * x * x
    scale = np.abs(ex).max()
    assert np.abs(fld[:, 0] - ex).max() < 1e-13 * scale
    assert max(np.abs(fld[:, 1] - gx).max(), np.abs(fld[:, 2] - gy).max(), np.abs(fld[:, 3] - gz).max()) < 2e-12 * scale
    # M f integrates the interpolant: 1^T M f == sum_q w f(q), and a cubic is NOT reproduced (the pin can fail)
    rp, ci = o.pattern(0)
    mf = np.add.reduceat(o.mass(0) * f[ci], rp[:-1])
    assert abs(mf.sum() - (w * ex).sum()) < 1e-12 * np.abs(w * ex).sum()
    fc = o.fields(X ** 3, 0)
    assert np.abs(fc[:, 0] - x ** 3).max() > 1e-4


# ------------------------------------------------------------------------------------------------ P5
def test_P5_rosenbluth_closed_forms_at_an_exterior_point(o3):
    from scipy import special
    n_s, theta = 1.3, 0.8
    o = o3.Oracle3V([dict(half=4.5, n=10, levels=0)], [dict(mass=1.0, charge=-1.0, grid=0)])
    x, y, z, w = o.ip_table(0)
    f = n_s * (math.pi * theta) ** -1.5 * np.exp(-(x * x + y * y + z * z) / theta)
    src = np.stack([f, -2 * x / theta * f, -2 * y / theta * f, -2 * z / theta * f], 1)
    pts = np.array([[7.0, 1.0, 2.0], [-6.0, 5.5, 0.5]])
    got = o.inner_at_points(0, [src], pts)
    for p, g in zip(pts, got):
        v = np.linalg.norm(p)
        vh = p / v
        xx = v / math.sqrt(theta)
        G = (special.erf(xx) - xx * 2 / math.sqrt(math.pi) * math.exp(-xx * xx)) / (2 * xx * xx)
        D = n_s / v * ((special.erf(xx) - G) * (np.eye(3) - np.outer(vh, vh)) + 2 * G * np.outer(vh, vh))
        Kv = -4 * n_s * G / theta * vh
        assert np.abs(_full(g[:6]) - D).max() < 3e-5 * np.abs(D).max()      # measured 8e-6 (quadrature of the Gaussian, h = 0.9)
        assert np.abs(g[6:] - Kv).max() < 1e-4 * np.abs(Kv).max()


# ------------------------------------------------------------------------------------------------ P6
def _state(o, species, temps, dens, drift):
    f = []
    for s, sp in enumerate(species):
        xyz = o.dof_coords(sp["grid"])
        th = temps[s] / sp["mass"]
        d = xyz - np.array(drift[s]) * math.sqrt(th)
        f.append(dens[s] * (math.pi * th) ** -1.5 * np.exp(-(d * d).sum(1) / th))
    return np.concatenate(f)


def test_P6_conservation_to_roundoff(o3):
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=4.0, charge=1.0, grid=1), dict(mass=9.0, charge=2.0, grid=1)]
    grids = [dict(half=4.0, n=4, levels=1), dict(half=2.0, n=3, levels=1)]
    o = o3.Oracle3V(grids, species)
    f = _state(o, species, [1.0, 1.4, 0.8], [1.0, 0.7, 0.2], [(0.1, -0.2, 0.3), (0.0, 0.2, -0.1), (-0.3, 0.0, 0.1)])
    rhs = o.apply(f)
    mom, scale = np.zeros(4), np.zeros(4)
    for s, sp in enumerate(species):
        xyz = o.dof_coords(sp["grid"])
        blk = rhs[o.f_off[s]:o.f_off[s + 1]]
        assert abs(blk.sum()) < 1e-12 * np.abs(blk).sum()                  # density of every species
        for k, psi in enumerate([xyz[:, 0], xyz[:, 1], xyz[:, 2], (xyz ** 2).sum(1)]):
            mom[k] += sp["mass"] * (psi @ blk)
            scale[k] += sp["mass"] * (np.abs(psi) @ np.abs(blk))
    assert np.all(np.abs(mom) < 1e-12 * scale)                             # three momenta and the energy
    assert np.abs(rhs).max() > 1e-6                                        # and the state is not an equilibrium
    # column sums of J vanish, apply == -(M/inf - J) f
    J = o.jacobian(f, float("inf"))
    for s, sp in enumerate(species):
        rp, ci = o.pattern(sp["grid"])
        v = J[o.v_off[s]:o.v_off[s + 1]]
        col = np.zeros(o.n_dof[sp["grid"]])
        np.add.at(col, ci, v)
        assert np.abs(col).max() < 1e-12 * np.abs(v).max()
        y = np.add.reduceat(v * f[o.f_off[s]:o.f_off[s + 1]][ci], rp[:-1])
        blk = rhs[o.f_off[s]:o.f_off[s + 1]]
        assert np.abs(blk + y).max() < 1e-12 * np.abs(blk).max()
    # the shift is the mass matrix: (M/dt - J) - (-J) = M/dt
    dt = 0.3
    A = o.jacobian(f, dt)
    for s, sp in enumerate(species):
        assert np.abs((A - J)[o.v_off[s]:o.v_off[s + 1]] - o.mass(sp["grid"]) / dt).max() < 1e-13 * np.abs(A).max()


# ------------------------------------------------------------------------------------------------ P8
def _lag2(x):
    return np.array([x * (x - 1) / 2, (1 - x) * (1 + x), x * (x + 1) / 2]), np.array([x - 0.5, -2 * x, x + 0.5])


def _global_basis_3d(half, n, refine_centre):
    """Geometric construction of the (nonconforming-mesh, conforming-space) Q2 space on n^3 cells of [-half, half]^3, with
    the cells whose closure contains the origin cut into 8 when `refine_centre`.  Column I of PH / PX / PY / PZ is the
    global shape function of free node I (and its derivatives) at the integration points.  A node of a small cell lying
    on a face or edge of a big cell without being one of its nodes carries no dof: the value there is the big cell's own
    interpolant (continuity).  Floating-point geometry, independent of the oracle's integer lattice."""
    h = 2 * half / n
    cells = []
    for ck in range(n):
        for cj in range(n):
            for ci in range(n):
                lo = np.array([-half + ci * h, -half + cj * h, -half + ck * h])
                if refine_centre and np.all(lo <= 1e-12) and np.all(lo + h >= -1e-12):
                    for b in range(8):
                        cells.append((lo + 0.5 * h * np.array([b & 1, (b >> 1) & 1, b >> 2]), h / 2, 1))
                else:
                    cells.append((lo, h, 0))
    key = lambda p: tuple(int(round((c + half) / h * 4)) for c in p)      # quarter-cell lattice holds every node
    nodes = {}
    for lo, hh, lev in cells:
        for a in range(27):
            p = lo + 0.5 * hh * np.array([a % 3, (a // 3) % 3, a // 9])
            nodes[key(p)] = p
    big = [c for c in cells if c[2] == 0]
    own = {id(c): {key(c[0] + 0.5 * c[1] * np.array([a % 3, (a // 3) % 3, a // 9])) for a in range(27)} for c in big}
    hanging = {}
    for lo, hh, lev in cells:
        if lev == 0:
            continue
        for a in range(27):
            p = lo + 0.5 * hh * np.array([a % 3, (a // 3) % 3, a // 9])
            for c in big:
                if np.all(p >= c[0] - 1e-12) and np.all(p <= c[0] + c[1] + 1e-12) and key(p) not in own[id(c)]:
                    hanging[key(p)] = c
    free = sorted((k for k in nodes if k not in hanging), key=lambda k: (k[2], k[1], k[0]))
    dof = {k: i for i, k in enumerate(free)}
    gx, gw = np.polynomial.legendre.leggauss(3)
    ip, w, PH, PX, PY, PZ = [], [], [], [], [], []
    for lo, hh, lev in cells:
        N = np.zeros((27, len(free)))
        for a in range(27):
            p = lo + 0.5 * hh * np.array([a % 3, (a // 3) % 3, a // 9])
            k = key(p)
            if k in dof:
                N[a, dof[k]] = 1.0
            else:
                c = hanging[k]
                v = [_lag2(-1 + 2 * (p[d] - c[0][d]) / c[1])[0] for d in range(3)]
                for b in range(27):
                    wgt = v[0][b % 3] * v[1][(b // 3) % 3] * v[2][b // 9]
                    if abs(wgt) > 1e-15:
                        N[a, dof[key(c[0] + 0.5 * c[1] * np.array([b % 3, (b // 3) % 3, b // 9]))]] += wgt
        for q in range(27):
            q1, q2, q3 = q % 3, (q // 3) % 3, q // 9
            (v1, d1), (v2, d2), (v3, d3) = _lag2(gx[q1]), _lag2(gx[q2]), _lag2(gx[q3])
            ip.append(lo + 0.5 * hh * (1 + np.array([gx[q1], gx[q2], gx[q3]])))
            w.append(gw[q1] * gw[q2] * gw[q3] * hh ** 3 / 8)
            val = lambda t1, t2, t3: np.einsum("k,j,i->kji", t3, t2, t1).ravel()
            PH.append(val(v1, v2, v3) @ N)
            PX.append(2 / hh * val(d1, v2, v3) @ N)
            PY.append(2 / hh * val(v1, d2, v3) @ N)
            PZ.append(2 / hh * val(v1, v2, d3) @ N)
    coords = np.array([nodes[k] for k in free])
    return np.array(ip), np.array(w), np.array(PH), np.array(PX), np.array(PY), np.array(PZ), coords


def test_P8_brute_force_dense_jacobian_with_hanging_nodes(o3):
    """Two species on two grids: a 3^3 grid with its centre cell refined (34 cells; 72 hanging nodes on faces and edges) and a
    uniform 2^3 grid.  Pins the fold P_e^T A_e P_e, the constrained field evaluation, the cross-grid inner integral, the
    species factors and the signs of the weak form."""
    dt = 0.7
    ext = [(2.0, 3, True), (1.0, 2, False)]
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=9.0, charge=2.0, grid=1)]
    o = o3.Oracle3V([dict(half=e[0], n=e[1], levels=1 if e[2] else 0) for e in ext], species)
    B = [_global_basis_3d(*e) for e in ext]
    for g in range(2):
        assert B[g][6].shape[0] == o.n_dof[g] and np.abs(B[g][6] - o.dof_coords(g)).max() < 1e-13   # same dofs, same order
        assert len(B[g][1]) == o.n_ip[g] and np.abs(B[g][2].sum(1) - 1).max() < 1e-13              # partition of unity
    assert o.n_cells[0] == 34 and o.n_dof[0] == 7 ** 3 + 26
    f = _state(o, species, [1.0, 1.5], [1.0, 0.6], [(0.2, -0.1, 0.3), (-0.2, 0.3, 0.1)])
    fs = [f[o.f_off[s]:o.f_off[s + 1]] for s in range(2)]
    vals, rhs = o.jacobian(f, dt), o.apply(f)
    for a, spa in enumerate(species):
        ga = spa["grid"]
        ipa, wa, PH, PX, PY, PZ, _ = B[ga]
        nq = len(ipa)
        D, Kv = np.zeros((nq, 3, 3)), np.zeros((nq, 3))
        for b, spb in enumerate(species):
            ipb, wb, QH, QX, QY, QZ, _ = B[spb["grid"]]
            nu = spa["charge"] ** 2 * spb["charge"] ** 2
            fj = QH @ fs[b]
            gj = np.stack([QX @ fs[b], QY @ fs[b], QZ @ fs[b]], 1)
            for i in range(nq):
                u = ipa[i][None, :] - ipb
                u2 = (u * u).sum(1)
                ok = u2 > 1e-20
                inv3 = np.where(ok, 1.0, 0.0) / np.where(ok, u2 ** 1.5, 1.0)
                U = (u2[:, None, None] * np.eye(3)[None] - u[:, :, None] * u[:, None, :]) * inv3[:, None, None]
                D[i] += nu / spa["mass"] ** 2 * np.einsum("j,jrc->rc", wb * fj, U)
                Kv[i] += nu / (spa["mass"] * spb["mass"]) * np.einsum("j,jrc,jc->r", wb, U, gj)
        n = PH.shape[1]
        A = np.zeros((n, n))
        for q in range(nq):
            gphi = np.stack([PX[q], PY[q], PZ[q]], 0)
            A += wa[q] * (np.outer(PH[q], PH[q]) / dt + gphi.T @ D[q] @ gphi - np.outer(gphi.T @ Kv[q], PH[q]))
        rp, ci = o.pattern(ga)
        dense = np.zeros((n, n))
        v = vals[o.v_off[a]:o.v_off[a + 1]]
        for i in range(n):
            dense[i, ci[rp[i]:rp[i + 1]]] = v[rp[i]:rp[i + 1]]
        assert np.linalg.norm(dense - A) < 1e-11 * np.linalg.norm(A)
        assert np.abs(dense - A).max() < 1e-11 * np.abs(A).max()
        assert np.all((np.abs(A) > 1e-13 * np.abs(A).max()) <= (dense != 0))     # the structural pattern holds every coupling
        Mq = (PH * wa[:, None]).T @ PH
        ref_rhs = (Mq / dt - A) @ fs[a]
        blk = rhs[o.f_off[a]:o.f_off[a + 1]]
        assert np.linalg.norm(blk - ref_rhs) < 1e-10 * np.linalg.norm(ref_rhs)


# ------------------------------------------------------------------------------------------------ P10
def test_P10_isotropization_rate_matches_appendix_B(o3):
    """dT_perp/dt = -(1/2) dT_par/dt = -nu_T (T_perp - T_par) for a bi-Maxwellian -- in 3V with
    T_par along z and T_perp in the (x, y) plane.  Same constant c_iso as the 2V pin: the Cartesian operator has the same
    normalisation as the gyro-averaged one."""
    g = TM.golden_rates(os.path.join(os.path.dirname(__file__), "golden", "nrl_rates.txt"))
    alpha = 1.3
    o = o3.Oracle3V([dict(half=3.6, n=8, levels=1)], [dict(mass=1.0, charge=-1.0, grid=0)])
    xyz = o.dof_coords(0)
    f = (1 / alpha) * math.pi ** -1.5 * np.exp(-(xyz[:, 2] ** 2 + (xyz[:, 0] ** 2 + xyz[:, 1] ** 2) / alpha))
    rhs = o.apply(f)
    rp, ci = o.pattern(0)
    mf = np.add.reduceat(o.mass(0) * f[ci], rp[:-1])
    n = mf.sum()
    tx, ty, tz = (2 * (xyz[:, d] ** 2) @ mf / n for d in range(3))
    dx, dy, dz = (2 * (xyz[:, d] ** 2) @ rhs / n for d in range(3))
    assert abs(n - 1) < 2e-3 and abs(tx / tz - alpha) < 1e-2 and abs(tx - ty) < 1e-12
    assert abs(dx + dy + dz) < 1e-12 * abs(dz)                              # energy
    assert abs(dx - dy) < 1e-12 * abs(dx)                                   # symmetry of the grid
    tperp, dperp = 0.5 * (tx + ty), 0.5 * (dx + dy)
    nu_t = TM.nrl_isotropization_rate(g["c_iso"], n, 1.0, tperp, tz)
    assert abs(-dperp / (tperp - tz) - nu_t) < 1.5e-2 * nu_t                # measured 7.5e-3 on this Q2 grid (h = 0.9 / 0.45)
