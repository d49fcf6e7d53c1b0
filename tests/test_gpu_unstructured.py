"""GPU parity on unstructured quadrilateral grids (landau_create_meshes) against the
oracle's unstructured path: same meshes, same seeded states.  Dofs are matched by coordinates (the order is each
implementation's own) and the CSR blocks compared as matrices; criterion as everywhere: relative Frobenius and
element-wise errors per (entry, species) block <= 1e-10."""
import numpy as np
import pytest

from paper_2209_03228_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def Bn():
    import torch
    assert torch.cuda.is_available()
    from paper_2209_03228_b200 import build
    build.build()
    from paper_2209_03228_b200 import binding
    binding.load()
    return binding


def _perm(a, b):
    p = np.array([int(np.argmin(((a - x) ** 2).sum(1))) for x in b])
    assert len(set(p)) == len(p) and np.abs(a[p] - b).max() < 1e-12
    return p


def _dense(rp, ci, v, n):
    A = np.zeros((n, n))
    for i in range(n):
        A[i, ci[rp[i]:rp[i + 1]]] = v[rp[i]:rp[i + 1]]
    return A


def _compare(L, o, vals, rhs, f_o, dt, entries):
    for b in entries:
        ref, ref_rhs = o.jacobian(f_o[b], dt), o.apply(f_o[b])
        for s in range(L.S):
            g = L.sgrid[s]
            n = int(L.n_dof[g])
            p = _perm(L.dof_coords(g), o.dof_coords(g))                 # L dof p[i] == oracle dof i
            A = _dense(*L.pattern(g), vals[b, L.v_off[s]:L.v_off[s + 1]], n)[np.ix_(p, p)]
            R = _dense(*o.pattern(g), ref[o.v_off[s]:o.v_off[s + 1]], n)
            assert np.linalg.norm(A - R) < TOL * np.linalg.norm(R) and np.abs(A - R).max() < TOL * np.abs(R).max()
            a, r = rhs[b, L.f_off[s]:L.f_off[s + 1]][p], ref_rhs[o.f_off[s]:o.f_off[s + 1]]
            assert np.linalg.norm(a - r) < TOL * np.linalg.norm(r) and np.abs(a - r).max() < TOL * np.abs(r).max()


@pytest.mark.parametrize("degree", [2, 3, 4])
@pytest.mark.parametrize("kernel", [0, 1])
def test_semicircle_two_species(orc, Bn, degree, kernel):
    import torch
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=25.0, charge=2.0, grid=1)]
    meshes = [W.semicircle_mesh(5.0, 2, 2), W.semicircle_mesh(1.0, 2, 1, core=0.6)]
    L = Bn.Landau.from_meshes(meshes, species, degree)
    o = orc.Oracle.from_meshes(meshes, species, degree)
    Bn.landau_set_inner_kernel(L.ctx, kernel)
    cfg = dict(index=82, species=species, state="shifted", alpha=[1.0, 1.0], batch=5)
    f_L = W.make_batch_f(cfg, [L.dof_coords(g) for g in range(2)], batch=5)
    f_o = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(2)], batch=5)
    dt = 0.5
    fd = torch.tensor(f_L, device="cuda")
    vals, rhs = L.jacobian(fd, dt).cpu().numpy(), L.apply(fd).cpu().numpy()
    _compare(L, o, vals, rhs, f_o, dt, [0, 4])
    # the slot-gather assembly agrees with the default one
    Bn.landau_set_assembly_kernel(L.ctx, 1)
    vals1 = L.jacobian(fd, dt).cpu().numpy()
    assert np.abs(vals1 - vals).max() < 1e-12 * np.abs(vals).max()
    # conservation on the GPU result: density per species, z-momentum, energy
    for b in range(5):
        mom, scale = np.zeros(2), np.zeros(2)
        for s, sp in enumerate(species):
            rz = L.dof_coords(sp["grid"])
            blk = rhs[b, L.f_off[s]:L.f_off[s + 1]]
            assert abs(blk.sum()) < 1e-12 * np.abs(blk).sum()
            for k, psi in enumerate([rz[:, 1], (rz ** 2).sum(1)]):
                mom[k] += sp["mass"] * (psi @ blk)
                scale[k] += sp["mass"] * (np.abs(psi) @ np.abs(blk))
        assert np.all(np.abs(mom) < 1e-12 * scale)
    L.close()


def test_paper_sized_semicircle_batch(orc, Bn):
    """24 Q3 cells per species (the 384 points of Table 13) for e- / D+, batch 256 through the many-column inner-integral
    kernel; the oracle checks sampled entries, every entry is checked for the mass identity."""
    import torch
    md = 3670.0
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=md, charge=1.0, grid=1)]
    meshes = [W.semicircle_mesh(5.0, 2, 2), W.semicircle_mesh(5.0 / np.sqrt(md), 2, 2)]
    L = Bn.Landau.from_meshes(meshes, species, 3)
    o = orc.Oracle.from_meshes(meshes, species, 3)
    cfg = dict(index=83, species=species, state="shifted", alpha=[1.0, 1.0], batch=256)
    f_L = W.make_batch_f(cfg, [L.dof_coords(g) for g in range(2)], batch=256)
    f_o = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(2)], batch=256)
    fd = torch.tensor(f_L, device="cuda")
    vals, rhs = L.jacobian(fd, 1.0).cpu().numpy(), L.apply(fd).cpu().numpy()
    _compare(L, o, vals, rhs, f_o, 1.0, [0, 101, 255])
    for s in range(2):
        tot = vals[:, L.v_off[s]:L.v_off[s + 1]].sum(1)                  # 1^T (M/dt - J) 1 = INT r dA (1^T J = 0)
        expect = o.mass(L.sgrid[s]).sum()
        assert np.abs(tot - expect).max() < 1e-9 * expect
    L.close()


def test_rectangles_as_a_mesh_equal_the_rectangular_path(Bn):
    """The same rectangular cells through landau_create_meshes and through landau_create: the per-point geometry path
    against the per-cell scale factors, on the GPU."""
    import torch
    cfg = W.tiny_config("uniform", 3, batch=3)
    meshes = []
    for g in cfg["grids"]:
        nr, nz = g["nr"], g["nz"]
        vr, vz = np.linspace(0, g["r_max"], nr + 1), np.linspace(g["z_min"], g["z_max"], nz + 1)
        v = np.array([(vr[i], vz[j]) for j in range(nz + 1) for i in range(nr + 1)])
        c = np.array([(j * (nr + 1) + i, j * (nr + 1) + i + 1, (j + 1) * (nr + 1) + i + 1, (j + 1) * (nr + 1) + i)
                      for j in range(nz) for i in range(nr)], dtype=np.int32)
        meshes.append((v, c))
    A = Bn.Landau(cfg["grids"], cfg["species"], 3)
    U = Bn.Landau.from_meshes(meshes, cfg["species"], 3)
    fa = W.make_batch_f(cfg, [A.dof_coords(g) for g in range(2)], batch=3)
    fu = W.make_batch_f(cfg, [U.dof_coords(g) for g in range(2)], batch=3)
    va = A.jacobian(torch.tensor(fa, device="cuda"), cfg["dt"]).cpu().numpy()
    vu = U.jacobian(torch.tensor(fu, device="cuda"), cfg["dt"]).cpu().numpy()
    for s in range(2):
        g = A.sgrid[s]
        n = int(A.n_dof[g])
        p = _perm(U.dof_coords(g), A.dof_coords(g))
        for b in range(3):
            Da = _dense(*A.pattern(g), va[b, A.v_off[s]:A.v_off[s + 1]], n)
            Du = _dense(*U.pattern(g), vu[b, U.v_off[s]:U.v_off[s + 1]], n)[np.ix_(p, p)]
            assert np.abs(Da - Du).max() < 1e-12 * np.abs(Da).max()
    A.close()
    U.close()


@pytest.mark.parametrize("degree", [2, 3, 4])
def test_triangles_two_species(orc, Bn, degree):
    """Simplex cells P2 - P4: two species on two triangle meshes of the half disc, Jacobian and operator
    application against the oracle, conservation on the GPU result; both inner-integral kernel families via the batch."""
    import torch
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=25.0, charge=2.0, grid=1)]
    meshes = [W.semicircle_triangles(5.0, 2, 2), W.semicircle_triangles(1.0, 2, 1, core=0.6)]
    L = Bn.Landau.from_meshes(meshes, species, degree)
    o = orc.Oracle.from_meshes(meshes, species, degree)
    cfg = dict(index=85, species=species, state="shifted", alpha=[1.0, 1.0], batch=9)
    f_L = W.make_batch_f(cfg, [L.dof_coords(g) for g in range(2)], batch=9)
    f_o = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(2)], batch=9)
    dt = 0.5
    fd = torch.tensor(f_L, device="cuda")
    vals, rhs = L.jacobian(fd, dt).cpu().numpy(), L.apply(fd).cpu().numpy()
    _compare(L, o, vals, rhs, f_o, dt, [0, 8])
    Bn.landau_set_inner_kernel(L.ctx, 1)
    vals1 = L.jacobian(fd[:2].contiguous(), dt).cpu().numpy()
    assert np.abs(vals1 - vals[:2]).max() < 1e-12 * np.abs(vals).max()
    for b in range(9):
        mom, scale = np.zeros(2), np.zeros(2)
        for s, sp in enumerate(species):
            rz = L.dof_coords(sp["grid"])
            blk = rhs[b, L.f_off[s]:L.f_off[s + 1]]
            assert abs(blk.sum()) < 1e-12 * np.abs(blk).sum()
            for k, psi in enumerate([rz[:, 1], (rz ** 2).sum(1)]):
                mom[k] += sp["mass"] * (psi @ blk)
                scale[k] += sp["mass"] * (np.abs(psi) @ np.abs(blk))
        assert np.all(np.abs(mom) < 1e-12 * scale)
    L.close()


def test_triangles_p4_batch_and_step(orc, Bn):
    """P4 on 48 triangles, e- / D+, batch 128 (many-column kernel), sampled entries against the oracle; then one
    backward-Euler step with landau_step (the batched solver on the triangle pattern) conserves density and energy."""
    import torch
    md = 3670.0
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=md, charge=1.0, grid=1)]
    meshes = [W.semicircle_triangles(5.0, 2, 2), W.semicircle_triangles(5.0 / np.sqrt(md), 2, 2)]
    L = Bn.Landau.from_meshes(meshes, species, 4)
    o = orc.Oracle.from_meshes(meshes, species, 4)
    assert L.n_ip[0] == 48 * 16
    cfg = dict(index=86, species=species, state="shifted", alpha=[1.0, 1.0], batch=128)
    f_L = W.make_batch_f(cfg, [L.dof_coords(g) for g in range(2)], batch=128)
    f_o = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(2)], batch=128)
    fd = torch.tensor(f_L, device="cuda")
    vals, rhs = L.jacobian(fd, 1.0).cpu().numpy(), L.apply(fd).cpu().numpy()
    _compare(L, o, vals, rhs, f_o, 1.0, [0, 127])
    u = fd[:4].clone()
    m_vals = L.jacobian(u, 1.0) - L.jacobian(u, float("inf"))
    before = L.spmv(m_vals, u).cpu().numpy()
    info = L.step(u, 0.05, newton_rtol=1e-11, max_newton=60, lin_rtol=1e-12, lin_max_it=2000)
    assert info["lin_failed"] == 0 and info["last_update"] <= 1e-11
    after = L.spmv(m_vals, u).cpu().numpy()
    for b in range(4):
        en0 = en1 = 0.0
        for s, sp in enumerate(species):
            rz = L.dof_coords(sp["grid"])
            sl = slice(L.f_off[s], L.f_off[s + 1])
            assert abs(after[b, sl].sum() - before[b, sl].sum()) < 1e-11 * abs(before[b, sl].sum())
            en0 += sp["mass"] * ((rz ** 2).sum(1) @ before[b, sl])
            en1 += sp["mass"] * ((rz ** 2).sum(1) @ after[b, sl])
        assert abs(en1 - en0) < 1e-9 * abs(en0)
    L.close()
