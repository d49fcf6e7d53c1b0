"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the same seeded
inputs.  Bar (BASELINE.json north_star): relative Frobenius error <= 1e-10 per (batch entry, species) block for
Jacobians and apply vectors; <= 1e-14 relative for the elliptic pieces; bit-exact for the integer CSR pattern.
"""
import math

import numpy as np
import pytest

from paper_2209_03228_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL = 1e-10


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


def _make(orc, Bn, cfg, nu=None):
    o = orc.Oracle(cfg["grids"], cfg["species"], cfg["degree"], nu=nu)
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"], nu=nu)
    return o, L


def _block_errors(L, got, ref, offs):
    """Per (entry, species) block: the larger of the relative Frobenius error (the north star's criterion, reading A14)
    and its element-wise companion max|a - r| / max|r| (so that a wrong small entry cannot hide under a large
    diagonal)."""
    errs = []
    for b in range(ref.shape[0]):
        for s in range(L.S):
            a, r = got[b, offs[s]:offs[s + 1]], ref[b, offs[s]:offs[s + 1]]
            errs.append(max(np.linalg.norm(a - r) / np.linalg.norm(r), np.abs(a - r).max() / np.abs(r).max()))
    return np.array(errs)


# ------------------------------------------------------------------------------------------------ pieces
def test_elliptic_pieces_device_accuracy(orc, Bn, torch_cuda):
    torch = torch_cuda
    ms, mps = [], []
    for e in np.linspace(-7, math.log10(0.5), 400):       # m from 1e-7 up
        ms.append(10 ** e); mps.append(1 - 10 ** e)
    for e in np.linspace(-7, math.log10(0.5), 400):       # m' from 1e-7 up (m -> 1)
        mps.append(10 ** e); ms.append(1 - 10 ** e)
    for m in np.linspace(0.55, 0.65, 101):                # across the branch split
        ms.append(m); mps.append(1 - m)
    m = torch.tensor(ms, dtype=torch.float64, device="cuda")
    mp = torch.tensor(mps, dtype=torch.float64, device="cuda")
    out = torch.empty(3 * len(ms), dtype=torch.float64, device="cuda")
    Bn.landau_ellip_eval(m, mp, out)
    got = out.cpu().numpy().reshape(-1, 3)
    worst = 0
    for k in range(len(ms)):
        e = orc.ellip(ms[k], mps[k])
        for c, name in enumerate(["P0", "Dc", "Q"]):
            worst = max(worst, abs(got[k, c] - e[name]) / e[name])
    assert worst < 1e-14, worst


def test_tensor_device_vs_oracle(orc, Bn, torch_cuda):
    torch = torch_cuda
    rng = np.random.default_rng(11)
    n = 4000
    r, rb = rng.uniform(1e-4, 5, n), rng.uniform(1e-4, 5, n)
    z, zb = rng.uniform(-5, 5, n), rng.uniform(-5, 5, n)
    near = rng.uniform(size=n) < 0.3
    rb[near] = r[near] * (1 + 1e-3 * rng.normal(size=near.sum()))
    zb[near] = z[near] + 1e-3 * rng.normal(size=near.sum())
    far = rng.uniform(size=n) < 0.3
    rb[far] *= 1e-3
    zb[far] *= 1e-3
    rb[:5], zb[:5] = r[:5], z[:5]                          # coincident pairs
    dev = [torch.tensor(a, dtype=torch.float64, device="cuda") for a in (r, z, rb, zb)]
    out = torch.empty(5 * n, dtype=torch.float64, device="cuda")
    Bn.landau_tensor_eval(*dev, out)
    got = out.cpu().numpy().reshape(n, 5)
    assert np.all(got[:5] == 0)
    worst = 0
    for k in range(5, n):
        ref, ok = orc.tensor(r[k], z[k], rb[k], zb[k])
        worst = max(worst, np.abs(got[k] - ref).max() / np.abs(ref).max())
    assert worst < 2e-14, worst


# ------------------------------------------------------------------------------------------------ small, full batch
@pytest.mark.parametrize("kind,degree", [("uniform", 2), ("uniform", 3), ("quadtree", 2), ("quadtree", 3), ("uniform", 4),
                                         ("quadtree", 4)])
@pytest.mark.parametrize("kernel", [1, 2, 3, 4, 5])
def test_tiny_jacobian_apply_and_coefficients(orc, Bn, torch_cuda, kind, degree, kernel):
    torch = torch_cuda
    cfg = W.tiny_config(kind, degree, batch=3)
    o, L = _make(orc, Bn, cfg)
    Bn.landau_set_inner_kernel(L.ctx, kernel)
    for g in range(o.G):   # bit-exact integer work + same dof convention
        rp, ci = L.pattern(g)
        rp2, ci2 = o.pattern(g)
        assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)
        assert np.abs(L.dof_coords(g) - o.dof_coords(g)).max() < 1e-14
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=3)
    fd = torch.tensor(f, device="cuda")
    vals = L.jacobian(fd, cfg["dt"]).cpu().numpy()
    ref = o.jacobian_batch(f, cfg["dt"])
    assert _block_errors(L, vals, ref, L.v_off).max() < TOL
    # the general slot-gather assembly kernel agrees with the default ring kernel (summation order differs only)
    Bn.landau_set_assembly_kernel(L.ctx, 1)
    vals1 = L.jacobian(fd, cfg["dt"]).cpu().numpy()
    Bn.landau_set_assembly_kernel(L.ctx, 0)
    assert _block_errors(L, vals1, ref, L.v_off).max() < TOL
    assert _block_errors(L, vals1, vals, L.v_off).max() < 1e-13
    # and so does the element-matrix + gather path that cells without a ring schedule take (forced here: 3 entries, ragged tile)
    Bn.landau_set_assembly_kernel(L.ctx, 3)
    vals3 = L.jacobian(fd, cfg["dt"]).cpu().numpy()
    Bn.landau_set_assembly_kernel(L.ctx, 0)
    assert _block_errors(L, vals3, ref, L.v_off).max() < TOL
    assert _block_errors(L, vals3, vals, L.v_off).max() < 1e-13
    # frozen coefficients D, K at the IPs (IP order is implementation-private: match by coordinates)
    with pytest.raises(Bn.LandauError):
        L.last_coefficients(4)                              # more entries than the last pass holds: refused, nothing copied
    dk = L.last_coefficients(3)
    for b in range(3):
        ref_dk = o.inner(f[b])
        for s in range(L.S):
            g = L.sgrid[s]
            r1, z1, _ = L.ip_table(g)
            r2, z2, _ = o.ip_table(g)
            p1, p2 = np.lexsort((r1, z1)), np.lexsort((r2, z2))
            a, r = dk[s][b].T[p1], ref_dk[s][p2]
            assert np.linalg.norm(a - r) < 1e-12 * np.linalg.norm(r)
    rhs = L.apply(fd).cpu().numpy()
    ref_rhs = o.apply_batch(f)
    assert _block_errors(L, rhs, ref_rhs, L.f_off).max() < TOL
    # conservation on the GPU result too
    for b in range(3):
        mom, scale = np.zeros(3), np.zeros(3)
        for s, sp in enumerate(cfg["species"]):
            rz = o.dof_coords(sp["grid"])
            blk = rhs[b, L.f_off[s]:L.f_off[s + 1]]
            assert abs(blk.sum()) < 1e-12 * np.abs(blk).sum()
            for k, psi in enumerate([rz[:, 1], rz[:, 0] ** 2 + rz[:, 1] ** 2]):
                mom[k] += sp["mass"] * np.dot(psi, blk)
                scale[k] += sp["mass"] * np.dot(np.abs(psi), np.abs(blk))
        assert abs(mom[0]) < 1e-12 * scale[0] and abs(mom[1]) < 1e-12 * scale[1]
    L.close()


def test_general_nu_matrix_path(orc, Bn, torch_cuda):
    """A nu matrix that is not rank one takes the per-species-column path."""
    torch = torch_cuda
    cfg = W.tiny_config("uniform", 2, batch=2)
    cfg["species"] = cfg["species"] + [dict(mass=9.0, charge=1.0, grid=1)]
    cfg["alpha"] = [1.0] * 3
    nu = np.array([[1.0, 4.0, 1.5], [4.0, 16.0, 3.0], [1.5, 3.0, 1.0]])
    o, L = _make(orc, Bn, cfg, nu=nu)
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=2)
    fd = torch.tensor(f, device="cuda")
    for kernel in (1, 2, 3, 4, 5):
        Bn.landau_set_inner_kernel(L.ctx, kernel)
        vals = L.jacobian(fd, 0.3).cpu().numpy()
        assert _block_errors(L, vals, o.jacobian_batch(f, 0.3), L.v_off).max() < TOL
        rhs = L.apply(fd).cpu().numpy()
        assert _block_errors(L, rhs, o.apply_batch(f), L.f_off).max() < TOL
    L.close()


def test_edge_cases_and_errors(orc, Bn, torch_cuda):
    torch = torch_cuda
    cfg = W.tiny_config("quadtree", 2, two_species=False, batch=1)
    o, L = _make(orc, Bn, cfg)
    f = W.make_batch_f(cfg, [o.dof_coords(0)], batch=1)
    fd = torch.tensor(f, device="cuda")
    # batch == 0 is a no-op
    out = torch.full((1, L.csr_stride), 7.0, dtype=torch.float64, device="cuda")
    Bn.landau_jacobian(L.ctx, fd, 0, 1.0, out)
    assert torch.all(out == 7.0)
    # dt = +inf gives -J;  M/dt - J - (-J) = M/dt
    a = L.jacobian(fd, 0.25).cpu().numpy()[0]
    b = L.jacobian(fd, float("inf")).cpu().numpy()[0]
    assert np.abs((a - b) - o.mass(0) / 0.25).max() < 1e-13 * np.abs(a).max()
    assert np.linalg.norm(b - o.jacobian(f[0], float("inf"))) < TOL * np.linalg.norm(b)
    # invalid arguments are reported, not executed
    with pytest.raises(Bn.LandauError):
        Bn.landau_jacobian(L.ctx, fd, 1, 0.0, out)
    with pytest.raises(Bn.LandauError):
        Bn.landau_jacobian(L.ctx, fd, -1, 1.0, out)
    with pytest.raises(Bn.LandauError):
        Bn.landau_create(cfg["grids"], cfg["species"], 5)
    with pytest.raises(Bn.LandauError):
        Bn.landau_create(cfg["grids"], [dict(mass=1.0, charge=-1.0, grid=3)], 2)
    # host-buffer entry points agree with the device ones, bit for bit
    hv = np.zeros((1, L.csr_stride))
    Bn.landau_jacobian_host(L.ctx, f, 1, 0.25, hv)
    assert np.array_equal(hv[0], a)
    hr = np.zeros((1, L.f_stride))
    Bn.landau_apply_host(L.ctx, f, 1, hr)
    assert np.array_equal(hr, L.apply(fd).cpu().numpy())
    # batch chunking does not change results
    cfg3 = W.tiny_config("uniform", 2, batch=5)
    o3, L3 = _make(orc, Bn, cfg3)
    f3 = torch.tensor(W.make_batch_f(cfg3, [o3.dof_coords(g) for g in range(o3.G)], batch=5), device="cuda")
    full = L3.jacobian(f3, 1.0).cpu().numpy()
    Bn.landau_set_batch_chunk(L3.ctx, 2)
    assert np.array_equal(L3.jacobian(f3, 1.0).cpu().numpy(), full)
    L.close()
    L3.close()


# ------------------------------------------------------------------------------------------------ BASELINE configs
def _sample_entries(B, seed):
    """first, last and ceil(log2 B) seeded entries (BASELINE.md CPU-baseline plan)."""
    rng = np.random.default_rng(seed)
    extra = rng.choice(B, size=min(B, max(1, math.ceil(math.log2(max(B, 2))))), replace=False)
    return sorted(set([0, B - 1] + [int(x) for x in extra]))


def _config_parity(orc, Bn, torch, cfg, B, entries, kernel=0, check_apply=True):
    o, L = _make(orc, Bn, cfg)
    Bn.landau_set_inner_kernel(L.ctx, kernel)
    coords = [L.dof_coords(g) for g in range(L.G)]
    for g in range(L.G):
        assert np.abs(coords[g] - o.dof_coords(g)).max() < 1e-14 * cfg["grids"][g]["r_max"]
    f = W.make_batch_f(cfg, coords, batch=B)
    fd = torch.tensor(f, device="cuda")
    vals = L.jacobian(fd, cfg["dt"])
    sub = vals[entries].cpu().numpy()
    ref = np.stack([o.jacobian(f[b], cfg["dt"]) for b in entries])
    errs = _block_errors(L, sub, ref, L.v_off)
    assert errs.max() < TOL, errs.max()
    # property that holds at any size: column sums of every J block vanish (1^T J = 0, conservation of density)
    J = L.jacobian(fd, float("inf"))
    for s in range(L.S):
        g = L.sgrid[s]
        _, ci = L.pattern(g)
        cid = torch.tensor(ci.astype(np.int64), device="cuda")
        blk = J[:, L.v_off[s]:L.v_off[s + 1]]
        colsum = torch.zeros((B, int(L.n_dof[g])), dtype=torch.float64, device="cuda").index_add_(1, cid, blk)
        colabs = torch.zeros((B, int(L.n_dof[g])), dtype=torch.float64, device="cuda").index_add_(1, cid, blk.abs())
        assert float(colsum.abs().max() / colabs.max()) < 1e-12
    if check_apply:
        rhs = L.apply(fd)[entries].cpu().numpy()
        ref_rhs = np.stack([o.apply(f[b]) for b in entries])
        assert _block_errors(L, rhs, ref_rhs, L.f_off).max() < TOL
    L.close()
    return errs.max()


def test_config1_full(orc, Bn, torch_cuda):
    _config_parity(orc, Bn, torch_cuda, W.config(1), 1, [0])
    _config_parity(orc, Bn, torch_cuda, W.config(1), 1, [0], kernel=2)


def test_config2_batch64(orc, Bn, torch_cuda):
    _config_parity(orc, Bn, torch_cuda, W.config(2), 64, _sample_entries(64, 2))


@pytest.mark.parametrize("B", [1, 16, 64, 256, 512])
def test_config3_ten_species(orc, Bn, torch_cuda, B):
    """BASELINE.json configs[2] names the sweep 1, 16, 64, 256, 512.  At 256 and 512 the ten-species / three-grid mix
    goes through the tiled-F store of K1 and the many-column K2 (stream mode at 512)."""
    _config_parity(orc, Bn, torch_cuda, W.config(3), B, _sample_entries(B, 3)[:4], check_apply=(B in (16, 256)))


@pytest.mark.parametrize("kernel", [2, 3, 4, 5])
@pytest.mark.parametrize("general_nu", [False, True])
def test_several_species_on_one_grid_forced_kernels(orc, Bn, torch_cuda, kernel, general_nu):
    """Three species on ONE grid + one on a second grid, forced through the tiled-F layouts of the many-column kernels
    (3: 16 x 128, 4: 16 x 256) and the plain layout (2): the species mix of K1 (rank-one nu) and the per-species columns
    (general nu) in every F layout, full batch against the oracle."""
    torch = torch_cuda
    cfg = W.tiny_config("quadtree", 3, batch=5)
    cfg["species"] = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=25.0, charge=1.0, grid=1),
                      dict(mass=50.0, charge=2.0, grid=1), dict(mass=100.0, charge=3.0, grid=1)]
    cfg["alpha"] = [1.0] * 4
    nu = None
    if general_nu:
        q2 = np.array([sp["charge"] ** 2 for sp in cfg["species"]])
        lnl = 1.0 + 0.05 * np.add.outer(np.arange(4), np.arange(4))      # symmetric, not rank one
        nu = np.outer(q2, q2) * lnl
    o, L = _make(orc, Bn, cfg, nu=nu)
    assert Bn.landau_is_separable(L.ctx) == (not general_nu)
    Bn.landau_set_inner_kernel(L.ctx, kernel)
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=5)
    fd = torch.tensor(f, device="cuda")
    vals = L.jacobian(fd, cfg["dt"]).cpu().numpy()
    assert _block_errors(L, vals, o.jacobian_batch(f, cfg["dt"]), L.v_off).max() < TOL
    rhs = L.apply(fd).cpu().numpy()
    assert _block_errors(L, rhs, o.apply_batch(f), L.f_off).max() < TOL
    L.close()


def test_host_buffer_path_in_pieces_against_oracle(orc, Bn, torch_cuda):
    """landau_jacobian_host cuts the batch into pieces (whole chunks, then the rest with its last part split off) and copies
    finished pieces on a second stream: config 2 with chunk 16 and B = 70 gives pieces 16, 16, 16, 16, 6; every sampled
    entry (one per piece + the seams) against the ORACLE, and the whole result against the one-call device path."""
    torch = torch_cuda
    cfg = W.config(2)
    B = 70
    o, L = _make(orc, Bn, cfg)
    Bn.landau_set_batch_chunk(L.ctx, 16)
    f = W.make_batch_f(cfg, [L.dof_coords(g) for g in range(L.G)], batch=B)
    hv = np.full((B, L.csr_stride), np.nan)
    Bn.landau_jacobian_host(L.ctx, f, B, cfg["dt"], hv)
    assert np.isfinite(hv).all()
    entries = [0, 15, 16, 40, 63, 64, 69]
    ref = np.stack([o.jacobian(f[b], cfg["dt"]) for b in entries])
    assert _block_errors(L, hv[entries], ref, L.v_off).max() < TOL
    Bn.landau_set_batch_chunk(L.ctx, 1024)
    dev = L.jacobian(torch.tensor(f, device="cuda"), cfg["dt"]).cpu().numpy()
    assert _block_errors(L, hv, dev, L.v_off).max() < 1e-13
    hr = np.full((B, L.f_stride), np.nan)
    Bn.landau_apply_host(L.ctx, f, B, hr)
    ref_rhs = np.stack([o.apply(f[b]) for b in entries])
    assert _block_errors(L, hr[entries], ref_rhs, L.f_off).max() < TOL
    L.close()


def test_host_buffer_path_large_split_against_oracle(orc, Bn, torch_cuda):
    """The 256-entry tail split of landau_jacobian_host (B >= 512 in the last chunk: pieces B - 256, 256) with pinned
    buffers, config 4 at B = 600 (pieces 344 + 256), sampled entries of both pieces against the oracle."""
    torch = torch_cuda
    cfg = W.config(4)
    B = 600
    o, L = _make(orc, Bn, cfg)
    f = torch.from_numpy(W.make_batch_f(cfg, [L.dof_coords(g) for g in range(L.G)], batch=B)).pin_memory()
    hv = torch.full((B, L.csr_stride), float("nan"), dtype=torch.float64).pin_memory()
    Bn.landau_jacobian_host(L.ctx, f, B, cfg["dt"], hv)
    hv = hv.numpy()
    assert np.isfinite(hv).all()
    entries = [0, 343, 344, 599]
    ref = np.stack([o.jacobian(f[b].numpy(), cfg["dt"]) for b in entries])
    assert _block_errors(L, hv[entries], ref, L.v_off).max() < TOL
    L.close()


def test_many_column_kernel_partial_wave_smaller_than_the_machine(orc, Bn, torch_cuda):
    """a 9 x 11 Q3 grid has 1584 integration points = 99 field-point tiles of 16; B = 600 gives 3 column
    tiles, T = 297 tiles on 148 SMs: the partial wave has ONE tile of 99 source-tile steps (< 148 CTAs).  Stream mode
    must not be taken for such a shape (empty shares); the result is checked against the oracle at both ends of the
    batch and in the middle column tile, and every block's column sums must vanish (a dropped tile would break both)."""
    torch = torch_cuda
    grid = dict(kind=0, r_max=5.0, z_min=-5.0, z_max=5.0, nr=9, nz=11, levels=0)
    cfg = dict(name="r_lt_p", index=96, grids=[grid], species=[dict(mass=1.0, charge=-1.0, grid=0)], degree=3, dt=0.5,
               batch=600, state="shifted", alpha=[1.0])
    _config_parity(orc, Bn, torch, cfg, 600, [0, 300, 599], check_apply=False)
    # same shape class with a general nu: two grids of 25 Q3 cells, three species per grid, B = 430 (1290 columns per
    # group: six column tiles of 256, T = 300 = 2 * 148 + 4, partial wave of 4 tiles x 25 steps = 100 steps < 148)
    g25 = dict(kind=0, r_max=5.0, z_min=-5.0, z_max=5.0, nr=5, nz=5, levels=0)
    g25b = dict(g25, r_max=1.0, z_min=-1.0, z_max=1.0)
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=2.0, charge=1.0, grid=0), dict(mass=3.0, charge=2.0, grid=0),
               dict(mass=25.0, charge=1.0, grid=1), dict(mass=30.0, charge=2.0, grid=1), dict(mass=40.0, charge=3.0, grid=1)]
    q2 = np.array([sp["charge"] ** 2 for sp in species])
    nu = np.outer(q2, q2) * (1.0 + 0.02 * np.add.outer(np.arange(6), np.arange(6)))
    cfg2 = dict(name="r_lt_p_general", index=95, grids=[g25, g25b], species=species, degree=3, dt=0.5, batch=430,
                state="shifted", alpha=[1.0] * 6)
    o = orc.Oracle(cfg2["grids"], species, 3, nu=nu)
    L = Bn.Landau(cfg2["grids"], species, 3, nu=nu)
    f = W.make_batch_f(cfg2, [L.dof_coords(g) for g in range(L.G)], batch=430)
    vals = L.jacobian(torch.tensor(f, device="cuda"), 0.5)
    entries = [0, 215, 429]
    ref = np.stack([o.jacobian(f[b], 0.5) for b in entries])
    assert _block_errors(L, vals[entries].cpu().numpy(), ref, L.v_off).max() < TOL
    L.close()


@pytest.mark.parametrize("cfg_no,B", [(4, 64), (4, 128), (3, 64), (2, 128)])
def test_stream_mode_with_fewer_tiles_than_resident_ctas(orc, Bn, torch_cuda, cfg_no, B):
    """The persistent many-column kernels cut their tiles along the source range also when there are FEWER tiles than
    resident CTAs (config 4: 208 field tiles on 2 x 148 CTAs of the 16 x 64 kernel, every tile is shared by two or three
    CTAs whose parts are added in part order) -- sampled entries against the oracle."""
    _config_parity(orc, Bn, torch_cuda, W.config(cfg_no), B, _sample_entries(B, cfg_no)[:3], check_apply=False)


def test_two_contexts_of_different_sizes_alternate(orc, Bn, torch_cuda):
    """the dynamic shared-memory limit of k3_ring / k4_tfqmr belongs to the device function, not to a
    context -- a small context created after a large one must not lower it."""
    torch = torch_cuda
    big, small = W.config(2), W.tiny_config("uniform", 2, batch=2)
    Lb = Bn.Landau(big["grids"], big["species"], big["degree"])
    Ls = Bn.Landau(small["grids"], small["species"], small["degree"])
    fb = torch.tensor(W.make_batch_f(big, [Lb.dof_coords(g) for g in range(Lb.G)], batch=2), device="cuda")
    fs = torch.tensor(W.make_batch_f(small, [Ls.dof_coords(g) for g in range(Ls.G)], batch=2), device="cuda")
    for _ in range(2):
        vb = Lb.jacobian(fb, 1.0)
        vs = Ls.jacobian(fs, 1.0)
        xb, itb, _ = Lb.solve(vb, fb, rtol=1e-8, max_it=400)
        xs, its, _ = Ls.solve(vs, fs, rtol=1e-8, max_it=400)
        torch.cuda.synchronize()
        assert int(itb.min()) > 0 and int(its.min()) > 0
    o = orc.Oracle(big["grids"], big["species"], big["degree"])
    ref = o.jacobian(fb[1].cpu().numpy(), 1.0)
    assert _block_errors(Lb, vb[1:2].cpu().numpy(), ref[None], Lb.v_off).max() < TOL
    Lb.close()
    Ls.close()


@pytest.mark.parametrize("degree,mode", [(4, 0), (3, 3)])
def test_reserve_covers_element_matrix_scratch(Bn, torch_cuda, degree, mode):
    """species that are not assembled by the ring kernel (Q4; any grid under assembly mode 3) keep their
    element matrices in a scratch buffer of their own, which landau_reserve must pre-size too: no allocation by the
    first landau_jacobian after it, and the same values as an unreserved context."""
    torch = torch_cuda
    cfg = W.tiny_config("quadtree", degree, batch=12)

    def make():
        L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
        Bn.landau_set_assembly_kernel(L.ctx, mode)
        return L
    L = make()
    fd = torch.tensor(W.make_batch_f(cfg, [L.dof_coords(g) for g in range(L.G)], batch=12), device="cuda")
    ref = L.jacobian(fd, cfg["dt"])                 # also loads every kernel the call takes (CUDA loads modules lazily)
    torch.cuda.synchronize()
    L.close()
    L = make()
    Bn.landau_reserve(L.ctx, 12)
    out = torch.empty_like(ref)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    Bn.landau_jacobian(L.ctx, fd, 12, cfg["dt"], out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    assert float((out - ref).norm() / ref.norm()) <= 1e-13
    L.close()


def test_non_blocking_stream_and_reserve(orc, Bn, torch_cuda):
    """scratch zeroing must be ordered on the caller's stream (torch.cuda.Stream() is non-blocking);
    landau_reserve pre-sizes the scratch so that the compute call allocates nothing."""
    torch = torch_cuda
    cfg = W.tiny_config("quadtree", 3, batch=40)
    o, L = _make(orc, Bn, cfg)
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=40)
    st = torch.cuda.Stream()
    fd = torch.tensor(f, device="cuda")
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        vals = L.jacobian(fd, cfg["dt"], stream=st.cuda_stream)    # first call: scratch grows, F zeroed on `st`
        rhs = L.apply(fd, stream=st.cuda_stream)
    st.synchronize()
    ref = o.jacobian_batch(f[[0, 39]], cfg["dt"])
    assert _block_errors(L, vals[[0, 39]].cpu().numpy(), ref, L.v_off).max() < TOL
    assert _block_errors(L, rhs[[0, 39]].cpu().numpy(), o.apply_batch(f[[0, 39]]), L.f_off).max() < TOL
    for B in (7, 1, 23):      # load every kernel variant the sizes below take (CUDA loads modules lazily)
        L.jacobian(fd[:B].contiguous(), cfg["dt"])
    torch.cuda.synchronize()
    L.close()
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    Bn.landau_reserve(L.ctx, 40)
    sizes = (40, 7, 1, 23)
    ins = [fd[:B].contiguous() for B in sizes]
    outs = [torch.empty((B, L.csr_stride), dtype=torch.float64, device="cuda") for B in sizes]
    rhss = [torch.empty((B, L.f_stride), dtype=torch.float64, device="cuda") for B in sizes]
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for B, fin, out, r in zip(sizes, ins, outs, rhss):
        Bn.landau_jacobian(L.ctx, fin, B, cfg["dt"], out)
        Bn.landau_apply(L.ctx, fin, B, r)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before          # the library allocated nothing after landau_reserve
    for out, r in zip(outs, rhss):
        assert _block_errors(L, out[:1].cpu().numpy(), ref[:1], L.v_off).max() < TOL
        assert _block_errors(L, r[:1].cpu().numpy(), o.apply_batch(f[:1]), L.f_off).max() < TOL
    L.close()


def test_config4_quadtree_bimaxwellian(orc, Bn, torch_cuda):
    _config_parity(orc, Bn, torch_cuda, W.config(4), 256, _sample_entries(256, 4)[:5])


def test_config6_paper_throughput_problem(orc, Bn, torch_cuda):
    """The paper's own 2V throughput problem (Table 5: ten species on three 14-cell quadtree Q3 grids,
    142 equations per species, batch 256) in the launch configuration `bench.py --advance` and BASELINE.md's context line
    are quoted on: Jacobian and operator application of the first, the last and seeded entries against the oracle."""
    cfg = W.config(6)
    assert cfg["batch"] == 256 and len(cfg["species"]) == 10 and len(cfg["grids"]) == 3
    _config_parity(orc, Bn, torch_cuda, cfg, 256, _sample_entries(256, 6))


def test_config5_bench_launch_configuration(orc, Bn, torch_cuda):
    """Full size of the bench workload (B = 1024, default chunking), sampled entries against the oracle."""
    _config_parity(orc, Bn, torch_cuda, W.config(5), 1024, [0, 517, 1023], check_apply=False)


def test_stream_mode_reproducible_and_batch_independent(Bn, torch_cuda):
    """Many-column K2 in persistent stream mode (config 3, B = 512: 384 tiles on 148 SMs): the same call gives the same
    bits, and an entry's Jacobian does not depend on the rest of the batch beyond summation order."""
    torch = torch_cuda
    cfg = W.config(3)
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    coords = [L.dof_coords(g) for g in range(L.G)]
    fd = torch.tensor(W.make_batch_f(cfg, coords, batch=512), device="cuda")
    a = L.jacobian(fd, cfg["dt"])
    b = L.jacobian(fd, cfg["dt"])
    assert torch.equal(a, b)
    c = L.jacobian(fd[:300].contiguous(), cfg["dt"])
    num = (c - a[:300]).norm(dim=1)
    assert float((num / a[:300].norm(dim=1)).max()) < 1e-13
    L.close()


def test_config5_maximum_batch(orc, Bn, torch_cuda):
    """BASELINE.json's largest size (config 5, B = 4096: 5.8 GB of CSR values, four passes of the default chunk): the
    first and the last entry against the oracle, every block's column sums, and the first pass bit-identical to a
    stand-alone run of the same 1024 entries."""
    torch = torch_cuda
    cfg = W.config(5)
    B = 4096
    o, L = _make(orc, Bn, cfg)
    coords = [L.dof_coords(g) for g in range(L.G)]
    f = W.make_batch_f(cfg, coords, batch=B)
    fd = torch.tensor(f, device="cuda")
    vals = L.jacobian(fd, cfg["dt"])
    entries = [0, B - 1]
    ref = np.stack([o.jacobian(f[b], cfg["dt"]) for b in entries])
    assert _block_errors(L, vals[entries].cpu().numpy(), ref, L.v_off).max() < TOL
    first = L.jacobian(fd[:1024].contiguous(), cfg["dt"])
    assert torch.equal(first, vals[:1024])
    del first
    vals.copy_(L.jacobian(fd, float("inf")))
    for s in range(L.S):
        g = L.sgrid[s]
        _, ci = L.pattern(g)
        cid = torch.tensor(ci.astype(np.int64), device="cuda")
        worst = 0.0
        for b0 in range(0, B, 512):
            blk = vals[b0:b0 + 512, L.v_off[s]:L.v_off[s + 1]]
            colsum = torch.zeros((blk.shape[0], int(L.n_dof[g])), dtype=torch.float64, device="cuda").index_add_(1, cid, blk)
            colabs = torch.zeros((blk.shape[0], int(L.n_dof[g])), dtype=torch.float64, device="cuda").index_add_(1, cid, blk.abs())
            worst = max(worst, float(colsum.abs().max() / colabs.max()))
        assert worst < 1e-12
    L.close()


def test_degenerate_cases(orc, Bn, torch_cuda):
    """Degenerate inputs of the method: (a) two species on two IDENTICAL grids -- every integration point of one grid
    coincides with one of the other, so the coincident-pair rule (reading A2) is exercised across grids; (b) a grid of
    a single cell; (c) a species that is absent (f = 0): its block must reduce to M/dt plus the field of the others."""
    torch = torch_cuda
    same = dict(kind=0, r_max=4.0, z_min=-4.0, z_max=4.0, nr=3, nz=5, levels=0)
    one = dict(kind=0, r_max=2.0, z_min=-2.0, z_max=2.0, nr=1, nz=1, levels=0)
    cfg = dict(name="degenerate", index=97, grids=[same, dict(same), one],
               species=[dict(mass=1.0, charge=-1.0, grid=0), dict(mass=2.0, charge=1.0, grid=1),
                        dict(mass=4.0, charge=2.0, grid=2)],
               degree=2, dt=0.3, batch=2, state="shifted", alpha=[1.0, 1.0, 1.0])
    o, L = _make(orc, Bn, cfg)
    f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=2)
    f[1, L.f_off[1]:L.f_off[2]] = 0.0                      # (c): species 1 absent in entry 1
    fd = torch.tensor(f, device="cuda")
    for kernel in (1, 2):
        Bn.landau_set_inner_kernel(L.ctx, kernel)
        vals = L.jacobian(fd, cfg["dt"]).cpu().numpy()
        assert _block_errors(L, vals, o.jacobian_batch(f, cfg["dt"]), L.v_off).max() < TOL
        rhs = L.apply(fd).cpu().numpy()
        ref = o.apply_batch(f)
        for b in range(2):
            for s in range(L.S):
                a, r = rhs[b, L.f_off[s]:L.f_off[s + 1]], ref[b, L.f_off[s]:L.f_off[s + 1]]
                assert np.linalg.norm(a - r) <= TOL * max(np.linalg.norm(r), 1e-300) or np.abs(r).max() == 0.0
    assert np.all(rhs[1, L.f_off[1]:L.f_off[2]] == 0.0)     # J[f] applied to f = 0 is exactly zero
    L.close()


def test_outputs_stay_inside_their_buffers(Bn, torch_cuda):
    """compute-sanitizer is not available on the pool: every output array is placed between two guard regions filled
    with a sentinel, and the guards must be untouched after jacobian (ring, gather and stream-mode paths), apply,
    spmv, solve and step."""
    torch = torch_cuda
    G = 4096
    sentinel = -7.25e300

    def guarded(rows, cols):
        buf = torch.full((rows * cols + 2 * G,), sentinel, dtype=torch.float64, device="cuda")
        return buf, buf[G:G + rows * cols].view(rows, cols)

    def intact(buf, rows, cols):
        return bool((buf[:G] == sentinel).all()) and bool((buf[G + rows * cols:] == sentinel).all())

    for cfg, B in ((W.tiny_config("quadtree", 3, batch=5), 5), (W.config(3), 300)):
        L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
        f = torch.tensor(W.make_batch_f(cfg, [L.dof_coords(g) for g in range(L.G)], batch=B), device="cuda")
        for asm in (0, 1, 3):
            Bn.landau_set_assembly_kernel(L.ctx, asm)
            vb, vals = guarded(B, L.csr_stride)
            Bn.landau_jacobian(L.ctx, f, B, cfg["dt"], vals)
            torch.cuda.synchronize()
            assert intact(vb, B, L.csr_stride) and bool(torch.isfinite(vals).all())
        Bn.landau_set_assembly_kernel(L.ctx, 0)
        rb, rhs = guarded(B, L.f_stride)
        Bn.landau_apply(L.ctx, f, B, rhs)
        yb, y = guarded(B, L.f_stride)
        Bn.landau_spmv(L.ctx, vals, f, B, y)
        xb, x = guarded(B, L.f_stride)
        x.zero_()
        Bn.landau_solve(L.ctx, vals, rhs, B, 1e-8, 100, x)
        ub, u = guarded(B, L.f_stride)
        u.copy_(f)
        Bn.landau_step(L.ctx, u, B, 1e-3, 1e-6, 3, 1e-8, 200)
        torch.cuda.synchronize()
        for buf in (rb, yb, xb, ub):
            assert intact(buf, B, L.f_stride)
        for t in (rhs, y, x, u):
            assert bool(torch.isfinite(t).all())
        L.close()
