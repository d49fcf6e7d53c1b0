"""The pieces of the C ABI composed into the paper's implicit advance (sec. 2.2): backward Euler with
the quasi-Newton iteration on the frozen-coefficient Jacobian,

    (M/dt - J[u]) delta = M (u^k - u)/dt + J[u] u,      u <- u + delta,

every operator application on the CUDA path (landau_jacobian, landau_apply, landau_spmv, landau_solve; torch only adds
vectors).  Checked against (a) the same iteration on the CPU oracle with direct solves and (b) what the paper states
for the converged step: density of every species, total z-momentum and total energy are conserved to the nonlinear
tolerance."""
import numpy as np
import pytest

from oracle import solve_oracle as SO
from paper_2209_03228_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _oracle_step(o, u0, dt, n_newton):
    """Backward-Euler step on the oracle: Newton with the sparse Jacobian, direct solves."""
    u = u0.copy()
    for _ in range(n_newton):
        a = o.jacobian(u, dt)
        ju = o.apply(u)
        delta = np.zeros_like(u)
        for s in range(o.S):
            g = o.sgrid[s]
            rp, ci = o.pattern(g)
            sl, vl = slice(o.f_off[s], o.f_off[s + 1]), slice(o.v_off[s], o.v_off[s + 1])
            rhs = SO.csr_matvec(rp, ci, o.mass(g), u0[sl] - u[sl]) / dt + ju[sl]
            delta[sl] = SO.solve_direct(rp, ci, a[vl], rhs)
        u = u + delta
    return u


@pytest.mark.parametrize("kind", ["uniform", "quadtree"])
def test_backward_euler_newton_step(orc, kind):
    import torch
    from paper_2209_03228_b200 import binding as Bn
    cfg = W.tiny_config(kind, 2, batch=2)
    # different temperatures and a drift so that the species exchange momentum and energy
    o = orc.Oracle(cfg["grids"], cfg["species"], cfg["degree"])
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    f0 = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=2)
    dt, n_newton = 0.1, 40
    u0 = torch.tensor(f0, device="cuda")
    m_vals = (L.jacobian(u0, 1.0) - L.jacobian(u0, float("inf")))          # CSR values of M
    u = u0.clone()
    for it in range(n_newton):
        a = L.jacobian(u, dt)
        rhs = L.spmv(m_vals, u0 - u) / dt + L.apply(u)
        delta, iters, _ = L.solve(a, rhs, rtol=1e-13, max_it=500)
        assert int(iters.min()) >= 0
        u = u + delta
    assert float(delta.norm() / u.norm()) < 1e-11                         # the Newton iteration has converged
    # (a) same step on the oracle
    got = u.cpu().numpy()
    for b in range(2):
        ref = _oracle_step(o, f0[b], dt, n_newton)
        for s in range(o.S):
            sl = slice(o.f_off[s], o.f_off[s + 1])
            assert np.linalg.norm(got[b, sl] - ref[sl]) < 1e-8 * np.linalg.norm(ref[sl])
    # (b) conservation over the step: moments psi^T M u with psi = 1, m z, m (r^2 + z^2)
    mu0, mu1 = L.spmv(m_vals, u0).cpu().numpy(), L.spmv(m_vals, u).cpu().numpy()
    for b in range(2):
        mom = np.zeros((2, 2))
        scale = np.zeros(2)
        for s, sp in enumerate(cfg["species"]):
            rz = o.dof_coords(sp["grid"])
            sl = slice(o.f_off[s], o.f_off[s + 1])
            n0, n1 = mu0[b, sl].sum(), mu1[b, sl].sum()
            assert abs(n1 - n0) < 1e-11 * abs(n0)                         # density of every species
            for k, psi in enumerate([rz[:, 1], rz[:, 0] ** 2 + rz[:, 1] ** 2]):
                mom[0, k] += sp["mass"] * (psi @ mu0[b, sl])
                mom[1, k] += sp["mass"] * (psi @ mu1[b, sl])
                scale[k] += sp["mass"] * (np.abs(psi) @ np.abs(mu0[b, sl]))
        assert abs(mom[1, 0] - mom[0, 0]) < 1e-10 * scale[0]              # total z-momentum
        assert abs(mom[1, 1] - mom[0, 1]) < 1e-10 * scale[1]              # total energy
        assert np.linalg.norm(got[b] - f0[b]) > 1e-4 * np.linalg.norm(f0[b])  # and the step is not trivial
    L.close()


def test_library_step_matches_composed_step_and_relaxes(orc):
    """landau_step (the same iteration inside the library, one inner integral per Newton iteration) against the oracle
    step; then several steps of an anisotropic state: densities, momentum and energy stay put while the distribution
    moves towards equilibrium (the relaxation experiment of PAPER.md sec. 6.1, qualitatively: || J[u] u || decreases)."""
    import torch
    from paper_2209_03228_b200 import binding as Bn
    cfg = W.tiny_config("uniform", 2, batch=2)
    o = orc.Oracle(cfg["grids"], cfg["species"], cfg["degree"])
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    f0 = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=2)
    dt = 0.1
    u = torch.tensor(f0, device="cuda")
    info = L.step(u, dt, newton_rtol=1e-12, max_newton=60, lin_rtol=1e-13, lin_max_it=500)
    assert info["lin_failed"] == 0 and info["last_update"] <= 1e-12 and 1 < info["newton_its"] < 60
    got = u.cpu().numpy()
    for b in range(2):
        ref = _oracle_step(o, f0[b], dt, info["newton_its"])
        for s in range(o.S):
            sl = slice(o.f_off[s], o.f_off[s + 1])
            assert np.linalg.norm(got[b, sl] - ref[sl]) < 1e-8 * np.linalg.norm(ref[sl])
    # a few more steps: invariants and relaxation
    u0 = torch.tensor(f0, device="cuda")
    m_vals = (L.jacobian(u0, 1.0) - L.jacobian(u0, float("inf")))
    def moments(v):
        mv = L.spmv(m_vals, v).cpu().numpy()
        out = []
        for b in range(2):
            dens, mom, en = [], 0.0, 0.0
            for s, sp in enumerate(cfg["species"]):
                rz = o.dof_coords(sp["grid"])
                blk = mv[b, o.f_off[s]:o.f_off[s + 1]]
                dens.append(blk.sum())
                mom += sp["mass"] * (rz[:, 1] @ blk)
                en += sp["mass"] * ((rz[:, 0] ** 2 + rz[:, 1] ** 2) @ blk)
            out.append((np.array(dens), mom, en))
        return out
    start = moments(u0)
    norms = [float(L.apply(u).norm())]
    for k in range(4):
        info = L.step(u, dt, newton_rtol=1e-12, max_newton=60, lin_rtol=1e-13, lin_max_it=500)
        assert info["lin_failed"] == 0 and info["last_update"] <= 1e-12
        norms.append(float(L.apply(u).norm()))
    end = moments(u)
    for b in range(2):
        assert np.abs(end[b][0] - start[b][0]).max() < 1e-10 * np.abs(start[b][0]).max()
        assert abs(end[b][2] - start[b][2]) < 1e-9 * abs(start[b][2])
        assert abs(end[b][1] - start[b][1]) < 1e-9 * abs(start[b][2])      # momentum, scaled by the energy
    assert all(n1 < n0 for n0, n1 in zip(norms, norms[1:])), norms          # || J[u] u || decreases: relaxation
    L.close()


def test_anisotropic_relaxation_history_against_nrl():
    """The relaxation experiment of PAPER.md sec. 6.1-6.2 in small: electrons start bi-Maxwellian (eq. 6.1,
    alpha = 1.3), 25 backward-Euler steps of landau_step to t = 0.5 t0.  Energy 2 T_perp + T_par is conserved to the
    nonlinear tolerance, the anisotropy decays monotonically, and its history follows the NRL rate
    equation of Appendix B -- closely at first, then slightly more slowly because the state stops being bi-Maxwellian
    (the discrepancy the paper reports under Fig. 5a)."""
    import math
    import torch
    from paper_2209_03228_b200 import binding as Bn
    grids = [dict(kind=0, r_max=5.0, z_min=-5.0, z_max=5.0, nr=8, nz=16, levels=0)]
    L = Bn.Landau(grids, [dict(mass=1.0, charge=-1.0, grid=0)], 3)
    rz = L.dof_coords(0)
    r, z = rz[:, 0], rz[:, 1]
    alpha, dt, nsteps = 1.3, 0.02, 25
    u = torch.tensor(((1 / alpha) * math.pi ** -1.5 * np.exp(-(z ** 2 + r ** 2 / alpha)))[None], device="cuda")
    m_vals = L.jacobian(u, 1.0) - L.jacobian(u, float("inf"))

    def temps(v):
        mv = L.spmv(m_vals, v).cpu().numpy()[0]
        return np.array([(r ** 2) @ mv, 2 * (z ** 2) @ mv]) / mv.sum()

    hist = [temps(u)]
    for k in range(nsteps):
        info = L.step(u, dt, newton_rtol=1e-11, max_newton=60, lin_rtol=1e-12, lin_max_it=1000)
        assert info["lin_failed"] == 0 and info["last_update"] <= 1e-11
        hist.append(temps(u))
    h = np.array(hist)
    energy = 2 * h[:, 0] + h[:, 1]
    assert np.abs(energy / energy[0] - 1).max() < 1e-10
    aniso = h[:, 0] - h[:, 1]
    assert np.all(np.diff(aniso) < 0)
    # NRL rate equation, RK4 (constant c_iso of tests/golden/nrl_rates.txt)
    c_iso = 2 ** 1.5 / math.sqrt(math.pi)

    def rate(y):
        a = y[0] / y[1] - 1
        nu = c_iso * y[1] ** -1.5 * (-3 + (a + 3) * math.atan(math.sqrt(a)) / math.sqrt(a)) / a ** 2
        return np.array([-nu * (y[0] - y[1]), 2 * nu * (y[0] - y[1])])

    y, nrl = h[0].copy(), [h[0][0] - h[0][1]]
    for k in range(nsteps):
        k1 = rate(y); k2 = rate(y + 0.5 * dt * k1); k3 = rate(y + 0.5 * dt * k2); k4 = rate(y + dt * k3)
        y = y + dt * (k1 + 2 * k2 + 2 * k3 + k4) / 6
        nrl.append(y[0] - y[1])
    nrl = np.array(nrl)
    assert abs(aniso[1] / nrl[1] - 1) < 5e-3           # first step: the state is still (almost) bi-Maxwellian
    assert 1.0 < aniso[-1] / nrl[-1] < 1.06            # later: slower than NRL, by a few per cent at t = 0.5 t0
    L.close()


def test_two_species_anisotropic_relaxation_against_nrl(orc):
    """The paper's verification experiment (sec. 6.1-6.2, Fig. 5a; App. B) with both species: a deuterium
    plasma, e- and D+ bi-Maxwellian by eq. (6.1) with alpha = 1.3 and T_e,par = 300, T_e,perp = 390, T_i,par = 200,
    T_i,perp = 260 eV (in units T0 = 300 eV), no shift, on quadtree-AMR Q3 grids of config-4 shape (4 x 8 base cells, 3
    levels towards the origin), each grid scaled to 5 initial parallel thermal speeds of its species.
    50 backward-Euler steps of landau_step to t = t0; the four temperatures (tests/temperature_moments.py) are compared
    with an RK4 integration of the coupled NRL equations: isotropisation of each species + thermal equilibration.

    * invariants: total energy to the nonlinear tolerance, density of each species to round-off;
    * ions (like-particle collisions dominate, electrons only heat them): anisotropy and heating follow NRL to 3 %;
    * electrons: at t = 0 the rate from the applied operator of the ORACLE (exact for this bi-Maxwellian state) is
      reproduced by the first step; the history is FASTER than the like-particle NRL rate because electron-ion
      pitch-angle scattering isotropises the electrons as well (Z = 1: comparable to e-e), and it stays monotone;
    * the first steps agree with the same steps on the oracle (direct solves) to 1e-8."""
    import math
    import os
    import torch
    import temperature_moments as TM
    from paper_2209_03228_b200 import binding as Bn
    g = TM.golden_rates(os.path.join(os.path.dirname(__file__), "golden", "nrl_rates.txt"))
    alpha, mi = 1.3, 3670.0
    mass, tau_par = [1.0, mi], [1.0, 200.0 / 300.0]
    theta = [tau_par[s] / mass[s] for s in range(2)]
    grids = [dict(kind=1, r_max=5.0 * math.sqrt(th), z_min=-5.0 * math.sqrt(th), z_max=5.0 * math.sqrt(th), nr=4, nz=8,
                  levels=3) for th in theta]
    species = [dict(mass=1.0, charge=-1.0, grid=0), dict(mass=mi, charge=1.0, grid=1)]
    L = Bn.Landau(grids, species, 3)
    o = orc.Oracle(grids, species, 3)
    rz = [L.dof_coords(s) for s in range(2)]
    f0 = np.concatenate([(1 / alpha) * (math.pi * theta[s]) ** -1.5 *
                         np.exp(-(rz[s][:, 1] ** 2 + rz[s][:, 0] ** 2 / alpha) / theta[s]) for s in range(2)])
    u = torch.tensor(f0[None], device="cuda")
    m_vals = L.jacobian(u, 1.0) - L.jacobian(u, float("inf"))

    def temps(v):
        mv = L.spmv(m_vals, v).cpu().numpy()[0]
        out = []
        for s in range(2):
            out += list(TM.temperatures(mv[L.f_off[s]:L.f_off[s + 1]], rz[s][:, 0], rz[s][:, 1], mass[s]))
        return np.array(out)                      # n_e, Te_perp, Te_par, n_i, Ti_perp, Ti_par

    dt, nsteps, n_oracle = 0.02, 50, 2
    hist, states = [temps(u)], []
    for k in range(nsteps):
        info = L.step(u, dt, newton_rtol=1e-11, max_newton=80, lin_rtol=1e-12, lin_max_it=2000)
        assert info["lin_failed"] == 0 and info["last_update"] <= 1e-11
        hist.append(temps(u))
        if k < n_oracle:
            states.append((u.cpu().numpy()[0].copy(), info["newton_its"]))
    h = np.array(hist)
    assert abs(h[0, 1] - 1.3) < 5e-3 and abs(h[0, 2] - 1.0) < 2e-3            # 390 / 300 eV, 300 / 300 eV
    assert abs(h[0, 4] - 260 / 300) < 5e-3 and abs(h[0, 5] - 200 / 300) < 2e-3
    # invariants
    energy = h[:, 0] * (2 * h[:, 1] + h[:, 2]) + h[:, 3] * (2 * h[:, 4] + h[:, 5])
    assert np.abs(energy / energy[0] - 1).max() < 1e-10
    assert np.abs(h[:, 0] / h[0, 0] - 1).max() < 1e-11 and np.abs(h[:, 3] / h[0, 3] - 1).max() < 1e-11
    # the same first steps on the oracle
    ref = f0
    for k in range(n_oracle):
        ref = _oracle_step(o, ref, dt, states[k][1])
        for s in range(2):
            sl = slice(o.f_off[s], o.f_off[s + 1])
            assert np.linalg.norm(states[k][0][sl] - ref[sl]) < 1e-8 * np.linalg.norm(ref[sl])
    # coupled NRL equations (App. B), y = (Te_perp, Te_par, Ti_perp, Ti_par), densities n = 1
    def rate(y):
        te, ti = (2 * y[0] + y[1]) / 3, (2 * y[2] + y[3]) / 3
        nub = TM.nrl_equilibration_rate(g["c_eq"], 1.0, 1.0, 1.0, mass[0], mass[1], te, ti)
        ne = TM.nrl_isotropization_rate(g["c_iso"], 1.0, mass[0], y[0], y[1])
        ni = TM.nrl_isotropization_rate(g["c_iso"], 1.0, mass[1], y[2], y[3])
        return np.array([-ne * (y[0] - y[1]) + nub * (ti - te), 2 * ne * (y[0] - y[1]) + nub * (ti - te),
                         -ni * (y[2] - y[3]) + nub * (te - ti), 2 * ni * (y[2] - y[3]) + nub * (te - ti)])
    nrl = TM.rk4(rate, h[0, [1, 2, 4, 5]], dt, nsteps)
    # ions
    ai, ai_nrl = h[:, 4] - h[:, 5], nrl[:, 2] - nrl[:, 3]
    assert np.all(np.diff(ai) < 0)
    assert np.abs((ai - ai[0])[1:] / (ai_nrl - ai[0])[1:] - 1).max() < 0.03
    ti, ti_nrl = (2 * h[:, 4] + h[:, 5]) / 3, (2 * nrl[:, 2] + nrl[:, 3]) / 3
    assert np.all(np.diff(ti) > 0)                                           # heated by the hotter electrons
    assert np.abs((ti - ti[0])[1:] / (ti_nrl - ti[0])[1:] - 1).max() < 0.03
    # electrons
    ae, ae_nrl = h[:, 1] - h[:, 2], nrl[:, 0] - nrl[:, 1]
    assert np.all(np.diff(ae) < 0)
    assert np.all(ae[1:] < ae_nrl[1:]) and ae[-1] > 0.4 * ae_nrl[-1]          # faster than like-particle NRL (e-i scattering)
    rhs0 = o.apply(f0)                                                      # exact initial rates from the oracle's operator
    rp, ci = o.pattern(0)
    mf = np.add.reduceat(o.mass(0) * f0[:o.f_off[1]][ci], rp[:-1])
    dperp, dpar = TM.temperature_rates(mf, rhs0[:o.f_off[1]], rz[0][:, 0], rz[0][:, 1], 1.0)
    assert dperp - dpar < -3 * TM.nrl_isotropization_rate(g["c_iso"], 1.0, 1.0, h[0, 1], h[0, 2]) * ae[0]   # e-e + e-i
    # backward Euler: M (u1 - u0)/dt = J[u1] u1, so the difference quotient of any moment IS that moment of the operator
    # applied to the new state (to the nonlinear tolerance), and it lies within 15 % of the initial rate
    rhs1 = L.apply(torch.tensor(states[0][0][None], device="cuda")).cpu().numpy()[0]
    mf1 = L.spmv(m_vals, torch.tensor(states[0][0][None], device="cuda")).cpu().numpy()[0]
    d1perp, d1par = TM.temperature_rates(mf1[:L.f_off[1]], rhs1[:L.f_off[1]], rz[0][:, 0], rz[0][:, 1], 1.0)
    fd = (ae[1] - ae[0]) / dt
    assert abs(fd / (d1perp - d1par) - 1) < 1e-7
    assert (dperp - dpar) < fd < 0 and abs(fd / (dperp - dpar) - 1) < 0.15
    L.close()


@pytest.mark.gpu
def test_step_reports_missing_convergence():
    """a step that stops at max_newton with the update above newton_rtol, or whose last linear solves missed
    lin_rtol, returns LANDAU_NOT_CONVERGED (u holds the last iterate) -- also to a caller that passes no info_host;
    the same step with enough iterations returns LANDAU_OK."""
    import ctypes as C
    import torch
    from paper_2209_03228_b200 import binding as Bn
    cfg = W.tiny_config("uniform", 2, batch=2)
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"])
    f0 = torch.tensor(W.make_batch_f(cfg, [L.dof_coords(g) for g in range(L.G)], batch=2), device="cuda")
    u = f0.clone()
    info = L.step(u, 0.1, newton_rtol=1e-12, max_newton=1, lin_rtol=1e-13, lin_max_it=500)       # one iteration is not enough
    assert not info["converged"] and info["newton_its"] == 1 and info["last_update"] > 1e-12 and info["lin_failed"] == 0
    assert bool(torch.isfinite(u).all()) and float((u - f0).norm()) > 0.0                          # the iterate was applied
    assert "not converged" in Bn.landau_last_error(L.ctx)
    u.copy_(f0)
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    rc = Bn.load().landau_step(L.ctx, C.c_void_p(u.data_ptr()), C.c_int(2), C.c_double(0.1), C.c_double(1e-12), C.c_int(1),
                               C.c_double(1e-13), C.c_int(500), None, st)                          # no info_host
    assert rc == Bn.LANDAU_NOT_CONVERGED == -5
    u.copy_(f0)
    info = L.step(u, 0.1, newton_rtol=1e-12, max_newton=60, lin_rtol=1e-13, lin_max_it=1)          # linear solves cut short
    assert not info["converged"] and info["lin_failed"] > 0
    u.copy_(f0)
    info = L.step(u, 0.1, newton_rtol=1e-12, max_newton=60, lin_rtol=1e-13, lin_max_it=500)
    assert info["converged"] and info["lin_failed"] == 0 and info["last_update"] <= 1e-12
    L.close()
