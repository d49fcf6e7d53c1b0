"""GPU parity of the 3V variant (include/landau3v.h) against the 3V oracle: same seeded inputs, element by element.
Criterion as for 2V (reading A14): per (entry, species) block the relative Frobenius error and its element-wise companion
max|a - r| / max|r|, both <= 1e-10; the frozen coefficients D, K alone <= 1e-12."""
import numpy as np
import pytest

from paper_2209_03228_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def o3():
    from oracle import oracle3v as O3
    O3.build()
    return O3


@pytest.fixture(scope="module")
def B3():
    import torch
    assert torch.cuda.is_available()
    from paper_2209_03228_b200 import build
    build.build()
    from paper_2209_03228_b200 import binding3v
    binding3v.load()
    return binding3v


def _block_errors(L, got, ref, offs):
    errs = []
    for b in range(ref.shape[0]):
        for s in range(L.S):
            a, r = got[b, offs[s]:offs[s + 1]], ref[b, offs[s]:offs[s + 1]]
            errs.append(max(np.linalg.norm(a - r) / np.linalg.norm(r), np.abs(a - r).max() / np.abs(r).max()))
    return np.array(errs)


@pytest.mark.parametrize("name", ["tiny", "tiny_uniform"])
@pytest.mark.parametrize("kernel", [1, 2, 3])
@pytest.mark.parametrize("general_nu", [False, True])
def test_tiny_parity(o3, B3, name, kernel, general_nu):
    import torch
    cfg = W.config3v(name, batch=5)
    nu = None
    if general_nu:   # symmetric, not rank one: one source column per (entry, species)
        nu = np.array([[1.0, 3.0], [3.0, 5.0]])
    L = B3.Landau3V(cfg["grids"], cfg["species"], nu=nu)
    o = o3.Oracle3V(cfg["grids"], cfg["species"], nu=nu)
    B3.landau3v_set_inner_kernel(L.ctx, kernel)
    f = W.make_batch_f3v(cfg, [o.dof_coords(g) for g in range(o.G)], batch=5)
    for g in range(L.G):
        assert np.abs(L.dof_coords(g) - o.dof_coords(g)).max() < 1e-14 * cfg["grids"][g]["half"]
    fd = torch.tensor(f, device="cuda")
    vals = L.jacobian(fd, cfg["dt"]).cpu().numpy()
    ref = o.jacobian_batch(f, cfg["dt"])
    assert _block_errors(L, vals, ref, L.v_off).max() < TOL
    # frozen coefficients at the integration points (IP order is implementation-private: match by coordinates)
    dk = L.last_coefficients(2)
    for b in range(2):
        ref_dk = o.inner(f[b])
        for s in range(L.S):
            g = L.sgrid[s]
            p1 = np.lexsort(np.stack(L.ip_table(g)[:3]))
            p2 = np.lexsort(np.stack(o.ip_table(g)[:3]))
            a, r = dk[s][b].T[p1], ref_dk[s][p2]
            assert np.linalg.norm(a - r) < 1e-12 * np.linalg.norm(r)
    rhs = L.apply(fd).cpu().numpy()
    assert _block_errors(L, rhs, o.apply_batch(f), L.f_off).max() < TOL
    # unshifted matrix, and the shift is exactly the mass matrix
    vinf = L.jacobian(fd, float("inf")).cpu().numpy()
    assert _block_errors(L, vinf, o.jacobian_batch(f, float("inf")), L.v_off).max() < TOL
    for s in range(L.S):
        m = o.mass(L.sgrid[s]) / cfg["dt"]
        blk = (vals - vinf)[:, L.v_off[s]:L.v_off[s + 1]]
        assert np.abs(blk - m[None]).max() < 1e-12 * np.abs(vals).max()
    # conservation on the GPU result: density per species, three momenta and energy -- needs the
    # symmetric nu both cases have
    for b in range(5):
        mom, scale = np.zeros(4), np.zeros(4)
        for s, sp in enumerate(cfg["species"]):
            xyz = o.dof_coords(sp["grid"])
            blk = rhs[b, L.f_off[s]:L.f_off[s + 1]]
            assert abs(blk.sum()) < 1e-12 * np.abs(blk).sum()
            for k, psi in enumerate([xyz[:, 0], xyz[:, 1], xyz[:, 2], (xyz ** 2).sum(1)]):
                mom[k] += sp["mass"] * (psi @ blk)
                scale[k] += sp["mass"] * (np.abs(psi) @ np.abs(blk))
        assert np.all(np.abs(mom) < 1e-12 * scale)
    L.close()


def test_batch_edges_chunks_and_host_buffers(o3, B3):
    import torch
    cfg = W.config3v("tiny", batch=13)
    L = B3.Landau3V(cfg["grids"], cfg["species"])
    o = o3.Oracle3V(cfg["grids"], cfg["species"])
    f = W.make_batch_f3v(cfg, [o.dof_coords(g) for g in range(o.G)], batch=13)
    fd = torch.tensor(f, device="cuda")
    whole = L.jacobian(fd, cfg["dt"]).cpu().numpy()                  # 13 columns: two n-tiles, the second ragged
    ref = o.jacobian_batch(f[[0, 7, 12]], cfg["dt"])
    assert _block_errors(L, whole[[0, 7, 12]], ref, L.v_off).max() < TOL
    B3.landau3v_set_batch_chunk(L.ctx, 4)                            # passes of 4, 4, 4, 1 entries
    chunked = L.jacobian(fd, cfg["dt"]).cpu().numpy()
    assert _block_errors(L, chunked, whole, L.v_off).max() < 1e-13   # summation order only (source range cut differently)
    assert _block_errors(L, chunked[[0, 7, 12]], ref, L.v_off).max() < TOL
    B3.landau3v_set_batch_chunk(L.ctx, 256)
    one = L.jacobian(fd[3:4].contiguous(), cfg["dt"]).cpu().numpy()  # a single entry: an 8-column tile with one column in use
    assert _block_errors(L, one, whole[3:4], L.v_off).max() < 1e-13
    # host buffers through the C ABI
    out_host = np.zeros((13, L.csr_stride))
    B3.landau3v_jacobian_host(L.ctx, f, 13, cfg["dt"], out_host)
    assert np.array_equal(out_host, L.jacobian(fd, cfg["dt"]).cpu().numpy())
    # batch 0 is a no-op, bad arguments are refused
    B3.landau3v_jacobian(L.ctx, fd, 0, cfg["dt"], torch.empty((0, L.csr_stride), dtype=torch.float64, device="cuda"))
    with pytest.raises(B3.LandauError):
        B3.landau3v_jacobian(L.ctx, fd, 13, 0.0, torch.empty((13, L.csr_stride), dtype=torch.float64, device="cuda"))
    with pytest.raises(B3.LandauError):
        L.last_coefficients(200)
    L.close()


def test_paper_sized_grids_batch_32(o3, B3):
    """e- / D+ on two of the paper's 3V grids (120 Q2 cells, 1,045 equations each) at the paper's batch size 32
    (Table 6), in the launch configuration bench.py times; the oracle checks sampled entries (first, last, one inside)."""
    import torch
    cfg = W.config3v("eD", batch=32)
    L = B3.Landau3V(cfg["grids"], cfg["species"])
    o = o3.Oracle3V(cfg["grids"], cfg["species"])
    assert L.n_cells[0] == 120 and L.n_dof[0] == 1045
    f = W.make_batch_f3v(cfg, [o.dof_coords(g) for g in range(o.G)], batch=32)
    fd = torch.tensor(f, device="cuda")
    vals = L.jacobian(fd, cfg["dt"]).cpu().numpy()
    rhs = L.apply(fd).cpu().numpy()
    pick = [0, 17, 31]
    assert _block_errors(L, vals[pick], o.jacobian_batch(f[pick], cfg["dt"]), L.v_off).max() < TOL
    assert _block_errors(L, rhs[pick], o.apply_batch(f[pick]), L.f_off).max() < TOL
    # properties that hold for every entry: finite, row sums of M/dt - J against 1 are the mass row sums (1^T J = 0 is a
    # column property; here: the block sum equals volume / dt)
    assert np.isfinite(vals).all()
    for s, sp in enumerate(cfg["species"]):
        vol = (2 * cfg["grids"][sp["grid"]]["half"]) ** 3
        tot = vals[:, L.v_off[s]:L.v_off[s + 1]].sum(1)
        assert np.abs(tot - vol / cfg["dt"]).max() < 1e-9 * vol / cfg["dt"]
    L.close()


def test_paper_problem_at_bench_launch_configuration(o3, B3):
    """The paper's 3V throughput problem exactly as `bench.py --config 7` runs it (Table 6: ten species on three
    120-cell Q2 grids, 1,045 equations per species, 9,720 integration points, batch 32): Jacobian and operator application
    of the first and the last entry against the oracle (about 1e9 long-double tensor evaluations per entry)."""
    import torch
    cfg = W.config3v("paper")
    assert cfg["batch"] == 32 and len(cfg["species"]) == 10
    L = B3.Landau3V(cfg["grids"], cfg["species"])
    o = o3.Oracle3V(cfg["grids"], cfg["species"])
    assert list(L.n_cells) == [120] * 3 and list(L.n_dof) == [1045] * 3 and int(sum(L.n_ip)) == 9720
    f = W.make_batch_f3v(cfg, [o.dof_coords(g) for g in range(o.G)], batch=32)
    fd = torch.tensor(f, device="cuda")
    vals = L.jacobian(fd, cfg["dt"])
    rhs = L.apply(fd)
    pick = [0, 31]
    assert _block_errors(L, vals[pick].cpu().numpy(), o.jacobian_batch(f[pick], cfg["dt"]), L.v_off).max() < TOL
    assert _block_errors(L, rhs[pick].cpu().numpy(), o.apply_batch(f[pick]), L.f_off).max() < TOL
    assert bool(torch.isfinite(vals).all()) and bool(torch.isfinite(rhs).all())
    L.close()


def test_ten_species_three_grids(o3, B3):
    """The paper's 3V throughput problem in small: ten species on three grids (several species per grid through the mixed
    source column), batch 2, against the oracle."""
    import torch
    cfg = W.config3v("paper", batch=2)
    grids = [dict(g, n=3, levels=1) for g in cfg["grids"]]           # 34 cells per grid keeps the oracle fast
    L = B3.Landau3V(grids, cfg["species"])
    o = o3.Oracle3V(grids, cfg["species"])
    f = W.make_batch_f3v(cfg, [o.dof_coords(g) for g in range(o.G)], batch=2)
    fd = torch.tensor(f, device="cuda")
    vals = L.jacobian(fd, cfg["dt"]).cpu().numpy()
    assert _block_errors(L, vals, o.jacobian_batch(f, cfg["dt"]), L.v_off).max() < TOL
    rhs = L.apply(fd).cpu().numpy()
    assert _block_errors(L, rhs, o.apply_batch(f), L.f_off).max() < TOL
    L.close()


def test_two_levels_and_general_nu_with_shared_grid(o3, B3):
    """Two nested refinement levels (constraint rows through two shells) and a non-rank-one nu with two species sharing a grid
    (one source column per (entry, species), zero outside the species' own grid), both inner-integral kernels."""
    import torch
    grids = [dict(half=3.0, n=2, levels=2), dict(half=1.0, n=3, levels=1)]
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=4.0, charge=1.0, grid=1), dict(mass=9.0, charge=2.0, grid=1)]
    nu = np.array([[1.0, 2.0, 0.5], [2.0, 3.0, 1.5], [0.5, 1.5, 4.0]])
    cfg = dict(index=97, species=species, state="shifted", alpha=[1.0] * 3, batch=9, dt=0.4)
    L = B3.Landau3V(grids, species, nu=nu)
    o = o3.Oracle3V(grids, species, nu=nu)
    assert L.n_cells[0] == 120                                          # 8 -> 64 -> 64 - 8 + 64
    f = W.make_batch_f3v(cfg, [o.dof_coords(g) for g in range(2)], batch=9)
    fd = torch.tensor(f, device="cuda")
    pick = [0, 8]
    ref, ref_rhs = o.jacobian_batch(f[pick], cfg["dt"]), o.apply_batch(f[pick])
    for kernel in (1, 2, 3):
        B3.landau3v_set_inner_kernel(L.ctx, kernel)
        vals, rhs = L.jacobian(fd, cfg["dt"]).cpu().numpy(), L.apply(fd).cpu().numpy()
        assert _block_errors(L, vals[pick], ref, L.v_off).max() < TOL
        assert _block_errors(L, rhs[pick], ref_rhs, L.f_off).max() < TOL
    # the first assembly version (every slot integrates its own entries) agrees with the default one
    B3.landau3v_set_assembly_kernel(L.ctx, 1)
    vals1 = L.jacobian(fd, cfg["dt"]).cpu().numpy()
    assert np.abs(vals1 - vals).max() < 1e-12 * np.abs(vals).max()
    L.close()
