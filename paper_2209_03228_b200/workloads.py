"""Seeded synthetic workloads shaped like BASELINE.json's configs.

This module serves BOTH the CUDA path and the oracle and therefore holds none of the method's arithmetic:
it only describes grids/species and samples analytic (bi-)Maxwellians at dof coordinates that the caller
obtained from whichever implementation it is driving.  Random numbers come from a counter-based
splitmix64 stream: value(seed, counter) -- no hidden state, so any subset of a batch can be regenerated.

Stand-ins: the paper's p4est AMR grids, Simmetrix meshes and PETSc option files are not
available; these generated grids and Maxwellian states replace them.
"""
import math

import numpy as np

SEED_BASE = 0x220903228000
_M64 = (1 << 64) - 1


def splitmix64(seed, counter):
    """Counter-based 64-bit hash: the `counter`-th output of a splitmix64 stream started at `seed`."""
    z = (seed + (counter + 1) * 0x9E3779B97F4A7C15) & _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def uniform01(seed, counter):
    return (splitmix64(seed, counter) >> 11) * (1.0 / (1 << 53))


def normal01(seed, counter):
    """Box-Muller on two sub-counters of `counter`."""
    u1 = uniform01(seed, 2 * counter + (1 << 40))
    u2 = uniform01(seed, 2 * counter + 1 + (1 << 40))
    return math.sqrt(-2.0 * math.log(1.0 - u1)) * math.cos(2.0 * math.pi * u2)


def _grid(kind, extent, nr, nz, levels=0):
    return dict(kind=kind, r_max=extent, z_min=-extent, z_max=extent, nr=nr, nz=nz, levels=levels)


_A = [2, 4, 7, 9, 12, 14, 16, 20, 40]
_Z = [1, 2, 3, 4, 6, 7, 8, 10, 18]


def config(index, batch=None):
    """Problem description of BASELINE.json configs[index-1] (index 1..5) plus small test-only variants.

    Returns dict(name, grids, species, degree, dt, batch, state) where state in {"maxwellian",
    "shifted", "bimaxwellian"} selects what `species_state` draws.
    """
    if index == 1:
        return dict(name="cfg1_e_8x16_Q2", index=1, grids=[_grid(0, 5.0, 8, 16)],
                    species=[dict(mass=1.0, charge=-1.0, grid=0)], degree=2, dt=1.0, batch=batch or 1,
                    state="maxwellian", alpha=[1.0])
    if index in (2, 5):
        n = (8, 16) if index == 2 else (14, 28)
        md = 3670.0
        return dict(name="cfg%d_eD_%dx%d_Q3" % (index, n[0], n[1]), index=index,
                    grids=[_grid(0, 5.0, n[0], n[1]), _grid(0, 5.0 / math.sqrt(md), n[0], n[1])],
                    species=[dict(mass=1.0, charge=-1.0, grid=0), dict(mass=md, charge=1.0, grid=1)],
                    degree=3, dt=1.0, batch=batch or (64 if index == 2 else 1024), state="shifted", alpha=[1.0, 1.0])
    if index == 3:
        masses = [1.0] + [1836.15 * a for a in _A]
        charges = [-1.0] + [float(z) for z in _Z]
        sgrid = [0, 1, 1, 1] + [2] * 6
        grids = [_grid(0, 5.0, 8, 8), _grid(0, 5.0 / math.sqrt(masses[1]), 8, 8),
                 _grid(0, 5.0 / math.sqrt(masses[4]), 8, 8)]
        return dict(name="cfg3_10species_3grids_Q3", index=3, grids=grids,
                    species=[dict(mass=m, charge=q, grid=g) for m, q, g in zip(masses, charges, sgrid)],
                    degree=3, dt=1.0, batch=batch or 256, state="maxwellian_nT", alpha=[1.0] * 10)
    if index == 4:
        md = 3670.0
        return dict(name="cfg4_eD_quadtree_Q3", index=4,
                    grids=[_grid(1, 5.0, 4, 8, 3), _grid(1, 5.0 / math.sqrt(md), 4, 8, 3)],
                    species=[dict(mass=1.0, charge=-1.0, grid=0), dict(mass=md, charge=1.0, grid=1)],
                    degree=3, dt=0.1, batch=batch or 256, state="bimaxwellian", alpha=[2.0, 0.5])
    if index == 6:
        # the paper's own throughput problem (Table 5): the ten species of config 3 on three
        # grids of 14 Q3 cells each (2 x 4 base cells, one refinement level at the origin: 142 equations per species),
        # batch 256, backward-Euler steps; not in BASELINE.json's list, used for the context line of BASELINE.md
        c3 = config(3)
        grids = [_grid(1, g["r_max"], 2, 4, 1) for g in c3["grids"]]
        # dt: the paper does not print it; 1e-3 t0 is the largest decade at which the quasi-Newton iteration on the sparse
        # Jacobian converges with the Z = 18 species present (nu ~ Z^4)
        return dict(name="paper_throughput_10species_3x14Q3", index=6, grids=grids, species=c3["species"], degree=3,
                    dt=1e-3, batch=batch or 256, state="maxwellian_nT", alpha=[1.0] * 10)
    raise ValueError("unknown config %r" % (index,))


def tiny_config(kind="uniform", degree=2, two_species=True, batch=2):
    """Small problems for fast tests (same recipe, fewer cells)."""
    if kind == "uniform":
        grids = [_grid(0, 5.0, 3, 6)] + ([_grid(0, 5.0 / 5.0, 2, 4)] if two_species else [])
    else:
        grids = [_grid(1, 5.0, 2, 4, 1)] + ([_grid(1, 5.0 / 5.0, 2, 4, 2)] if two_species else [])
    species = [dict(mass=1.0, charge=-1.0, grid=0)]
    if two_species:
        species.append(dict(mass=25.0, charge=2.0, grid=1))
    return dict(name="tiny_%s_Q%d" % (kind, degree), index=90 + degree, grids=grids, species=species, degree=degree,
                dt=0.5, batch=batch, state="shifted", alpha=[1.0] * len(species))


def species_state(cfg, batch=None, entries=None):
    """Seeded (n, T, u, alpha) per (entry, species): arrays [len(entries), S].  Draw order (entry, species, {n,T,u})."""
    B = batch or cfg["batch"]
    entries = list(range(B)) if entries is None else list(entries)
    S = len(cfg["species"])
    seed = SEED_BASE + cfg["index"]
    n = np.ones((len(entries), S))
    T = np.ones((len(entries), S))
    u = np.zeros((len(entries), S))
    al = np.tile(np.asarray(cfg["alpha"], dtype=np.float64), (len(entries), 1))
    st = cfg["state"]
    for row, b in enumerate(entries):
        for s in range(S):
            c = (b * S + s) * 3
            theta_ref = 1.0 / cfg["species"][s]["mass"]
            if st in ("shifted", "maxwellian_nT"):
                n[row, s] = 0.9 + 0.2 * uniform01(seed, c)
                T[row, s] = 0.8 + 0.4 * uniform01(seed, c + 1)
                if st == "shifted":
                    u[row, s] = 0.05 * math.sqrt(theta_ref) * normal01(seed, c + 2)
            elif st == "bimaxwellian":
                n[row, s] = 0.9 + 0.2 * uniform01(seed, c)
                T[row, s] = 0.9 + 0.2 * uniform01(seed, c + 1)
    return n, T, u, al


def sample_state(mass, n, T, u, alpha, rz):
    """f = (n/alpha)(pi theta)^{-3/2} exp(-((z-u)^2 + r^2/alpha)/theta), theta = T/mass (eq. 6.1, reading A11)."""
    theta = T / mass
    r, z = rz[:, 0], rz[:, 1]
    return (n / alpha) * (math.pi * theta) ** -1.5 * np.exp(-((z - u) ** 2 + r * r / alpha) / theta)


def sample_state_grad(mass, n, T, u, alpha, rz):
    """Analytic (f, df/dr, df/dz) of the same state (used by closed-form pins only)."""
    theta = T / mass
    r, z = rz[:, 0], rz[:, 1]
    f = sample_state(mass, n, T, u, alpha, rz)
    return f, f * (-2.0 * r / (alpha * theta)), f * (-2.0 * (z - u) / theta)


def make_batch_f(cfg, dof_coords, batch=None, entries=None):
    """Nodal interpolant of the seeded states: array [len(entries), sum_alpha n_dof(g(alpha))].

    dof_coords[g] = [n_dof_g, 2] (r, z) from the implementation being driven.
    """
    n, T, u, al = species_state(cfg, batch, entries)
    out = []
    for row in range(n.shape[0]):
        parts = []
        for s, sp in enumerate(cfg["species"]):
            parts.append(sample_state(sp["mass"], n[row, s], T[row, s], u[row, s], al[row, s], dof_coords[sp["grid"]]))
        out.append(np.concatenate(parts))
    return np.ascontiguousarray(np.stack(out))


# ------------------------------------------------------------------------------------------------------------------
# 3V workloads (Table 6): Q2 hexahedra on cubes [-half, half]^3
# ------------------------------------------------------------------------------------------------------------------
def _grid3(half, n, levels=0):
    return dict(half=half, n=n, levels=levels)


def config3v(name="paper", batch=None):
    """3V problem descriptions.

    "paper": the paper's 3V throughput problem (Table 6: batch 32) -- the ten species of config 3
             (electrons, deuterium, eight heavier ions) on three grids of 120 Q2 cells each (4 x 4 x 4 base cells, one
             refinement level about the origin: 1,045 equations per species), each grid scaled to 5 thermal speeds of
             its lightest species;
    "eD":    e- / D+ on two such grids (the 3V analogue of config 2), shifted Maxwellians;
    "tiny" / "tiny_uniform": two species on small grids (3^3 base cells with the centre cell refined + 2^3 cells;
             uniform 3^3 + 2^3) for fast tests.
    The `state` recipes are those of the 2V configs (species_state); a drift is along z.
    """
    if name == "paper":
        c3 = config(3)
        lightest = {0: 1.0, 1: c3["species"][1]["mass"], 2: c3["species"][4]["mass"]}
        grids = [_grid3(5.0 / math.sqrt(lightest[g]), 4, 1) for g in range(3)]
        return dict(name="paper_3V_10species_3x120Q2", index=7, dim=3, grids=grids, species=c3["species"], dt=1e-3,
                    batch=batch or 32, state="maxwellian_nT", alpha=[1.0] * 10)
    if name == "eD":
        md = 3670.0
        return dict(name="3V_eD_2x120Q2", index=8, dim=3, grids=[_grid3(5.0, 4, 1), _grid3(5.0 / math.sqrt(md), 4, 1)],
                    species=[dict(mass=1.0, charge=-1.0, grid=0), dict(mass=md, charge=1.0, grid=1)], dt=1.0,
                    batch=batch or 32, state="shifted", alpha=[1.0, 1.0])
    if name in ("tiny", "tiny_uniform"):
        lev = 1 if name == "tiny" else 0
        return dict(name="3V_" + name, index=95 + lev, dim=3, grids=[_grid3(4.0, 3, lev), _grid3(4.0 / 3.0, 2, 0)],
                    species=[dict(mass=1.0, charge=-1.0, grid=0), dict(mass=9.0, charge=2.0, grid=1)], dt=0.5,
                    batch=batch or 3, state="shifted", alpha=[1.0, 1.0])
    raise ValueError("unknown 3V config %r" % (name,))


def sample_state3v(mass, n, T, u, alpha, xyz):
    """The state of sample_state in Cartesian coordinates: r^2 = x^2 + y^2, z parallel."""
    theta = T / mass
    return (n / alpha) * (math.pi * theta) ** -1.5 * np.exp(-((xyz[:, 2] - u) ** 2 + (xyz[:, 0] ** 2 + xyz[:, 1] ** 2) / alpha) / theta)


def make_batch_f3v(cfg, dof_coords, batch=None, entries=None):
    """Nodal interpolant of the seeded states on 3V grids: dof_coords[g] = [n_dof_g, 3] (x, y, z)."""
    n, T, u, al = species_state(cfg, batch, entries)
    out = []
    for row in range(n.shape[0]):
        out.append(np.concatenate([sample_state3v(sp["mass"], n[row, s], T[row, s], u[row, s], al[row, s], dof_coords[sp["grid"]])
                                   for s, sp in enumerate(cfg["species"])]))
    return np.ascontiguousarray(np.stack(out))


# ------------------------------------------------------------------------------------------------------------------
# unstructured quadrilateral meshes (sec. 5.2, Fig. 4: "semi-circular grids ... with
# tensor elements").  The paper's mesh files are not available; this generator stands in for them.
# ------------------------------------------------------------------------------------------------------------------
def semicircle_mesh(radius, n=2, m=2, core=0.5):
    """Straight-sided quadrilateral mesh of the half disc r >= 0, r^2 + z^2 <= radius^2 (polygonal boundary): a core
    rectangle [0, a] x [-a, a], a = core * radius / sqrt(2), of n x 2n cells, and a ring of 4n x m cells between its
    three outer sides and the circle (an O-grid).  n = 2, m = 2 gives 24 cells -- with Q3 the 384 integration points of the
    paper's Table 13.  Returns (vertices [nv, 2] as (r, z), cells [nc, 4] counter-clockwise vertex ids).
    Input description only: no arithmetic of the method lives here."""
    a = core * radius / math.sqrt(2.0)
    verts, index = [], {}

    def vid(key, r, z):
        if key not in index:
            index[key] = len(verts)
            verts.append((r, z))
        return index[key]

    h = a / n
    for j in range(2 * n + 1):
        for i in range(n + 1):
            vid(("c", i, j), i * h, -a + j * h)
    cells = []
    for j in range(2 * n):
        for i in range(n):
            cells.append((index[("c", i, j)], index[("c", i + 1, j)], index[("c", i + 1, j + 1)], index[("c", i, j + 1)]))
    # perimeter of the core from (0, -a) along the bottom, up the right side and back along the top to (0, a)
    per = [("c", i, 0) for i in range(n + 1)] + [("c", n, j) for j in range(1, 2 * n + 1)] + [("c", i, 2 * n) for i in range(n - 1, -1, -1)]
    K = len(per) - 1   # 4 n edges
    for k, key in enumerate(per):
        p = verts[index[key]]
        th = -0.5 * math.pi + math.pi * k / K
        c = (radius * math.cos(th) if 0 < k < K else 0.0, radius * math.sin(th))
        for l in range(1, m + 1):
            t = l / m
            vid(("r", k, l), p[0] + t * (c[0] - p[0]), p[1] + t * (c[1] - p[1]))

    def ring(k, l):
        return index[per[k]] if l == 0 else index[("r", k, l)]

    for k in range(K):
        for l in range(m):
            # (k, l) -> (k, l+1) -> (k+1, l+1) -> (k+1, l) runs counter-clockwise in the (r, z) plane
            cells.append((ring(k, l), ring(k, l + 1), ring(k + 1, l + 1), ring(k + 1, l)))
    return np.array(verts, dtype=np.float64), np.array(cells, dtype=np.int32)


def semicircle_triangles(radius, n=2, m=2, core=0.5):
    """The cells of semicircle_mesh cut along a diagonal: a conforming triangle mesh of the same half disc (stand-in for the
    paper's Simmetrix meshes, sec. 5.1).  Returns (vertices [nv, 2], cells [2 nc, 3] counter-clockwise)."""
    v, q = semicircle_mesh(radius, n, m, core)
    tri = []
    for c in q:
        tri.append((c[0], c[1], c[2]))
        tri.append((c[0], c[2], c[3]))
    return v, np.array(tri, dtype=np.int32)
