"""Seeded synthetic inputs for the qNEP force-evaluation path (arXiv 2601.19034).

This module serves BOTH the fp64 oracle (``oracle/``) and the CUDA path
(``paper_2601_19034_b200/``).  It holds none of the method's arithmetic: it
only places atoms, draws random model parameters and names the electrostatics
settings of each BASELINE.json config.  The one model quantity that depends
on the method -- the descriptor scaler ``s_nu`` -- is read
from ``scalers.json``, a table written by the committed script
``oracle/make_scalers.py`` which calls only ``oracle/``.

The paper's datasets and trained models
are not available; these structures stand in for them and take their species
counts, densities and cell sizes.

Conventions
-----------
* positions: float64 ``[3][N]`` component-major (the C-ABI layout), Angstrom.
* types: int32 ``[N]``.
* box: float64 ``[9]``, rows are the cell vectors (orthorhombic in all configs).
* params: float32 flat vector in the documented order (include/qnep.h):
  ``c_R[ti][tj][n][k]``, ``c_A[ti][tj][n][k]``, ``s[D]``, then per type
  ``w0[H][D], b0[H], w1U[H], w1q[H]``, then ``b1U, b1q``.
"""
from __future__ import annotations

import json
import os
from dataclasses import dataclass, field

import numpy as np
from scipy.spatial import cKDTree

BASE_SEED = 20260119  # seeds are BASE_SEED + config index

_HERE = os.path.dirname(os.path.abspath(__file__))


# ----------------------------------------------------------------------------
# plain-data descriptions (mirrors of the C structs in include/qnep.h)
# ----------------------------------------------------------------------------
@dataclass
class ModelDesc:
    n_types: int
    n_max_r: int = 4
    n_max_a: int = 4
    l_max: int = 4
    basis_r: int = 8          # S3: k = 0..basis -> basis+1 Chebyshev functions
    basis_a: int = 8
    n_neurons: int = 80
    rc_r: float = 6.0
    rc_a: float = 4.0
    mode: int = 2             # 1: U^r+U^k+U^s (Eq. 3); 2: U^k only (Eq. 5)
    sqrt_eps_inf: float = 1.5  # S15
    q_total: float = 0.0
    l_max_4b: int = 0         # 2: NEP4 4-body terms on (one descriptor per angular radial channel; reading Z2)
    l_max_5b: int = 0         # 1: NEP4 5-body terms on

    @property
    def n_desc(self) -> int:
        return ((self.n_max_r + 1) + (self.n_max_a + 1) * self.l_max
                + ((self.n_max_a + 1) if self.l_max_4b == 2 else 0) + ((self.n_max_a + 1) if self.l_max_5b == 1 else 0))

    def n_params(self) -> int:
        T, H, D = self.n_types, self.n_neurons, self.n_desc
        nr = T * T * (self.n_max_r + 1) * (self.basis_r + 1)
        na = T * T * (self.n_max_a + 1) * (self.basis_a + 1)
        return nr + na + D + T * (H * D + 3 * H) + 2


@dataclass
class EsDesc:
    method: int = 2           # 0 none, 1 Ewald, 2 PPPM
    alpha: float = 0.3
    ewald_nmax2: int = 64     # S7: keep integer n.n <= nmax2
    grid: tuple = (32, 32, 32)
    order: int = 5


@dataclass
class Workload:
    name: str
    pos: np.ndarray           # float64 [3][N]
    types: np.ndarray         # int32 [N]
    box: np.ndarray           # float64 [9]
    model: ModelDesc
    params: np.ndarray        # float32 [n_params]
    es: EsDesc
    masses: np.ndarray = field(default=None)  # amu per type (MD only)
    zbl: tuple = None         # optional ZBL core: (r_inner, r_outer, Z per species) (reading Z1)
    extra: dict = field(default_factory=dict)

    @property
    def n_atoms(self) -> int:
        return int(self.types.shape[0])


# ----------------------------------------------------------------------------
# model parameters
# ----------------------------------------------------------------------------
def load_scaler(key: str, n_desc: int) -> np.ndarray:
    """Frozen descriptor scaler s_nu for a structure family (S5)."""
    path = os.path.join(_HERE, "scalers.json")
    if os.path.exists(path):
        with open(path) as f:
            table = json.load(f)
        if key in table and len(table[key]) == n_desc:
            return np.asarray(table[key], dtype=np.float64)
    # No table yet (only the case while oracle/make_scalers.py runs): unit scaler.
    return np.ones(n_desc, dtype=np.float64)


def random_params(model: ModelDesc, seed: int, scaler: np.ndarray | None = None) -> np.ndarray:
    """Random-init qNEP parameters (BASELINE.json configs).

    c ~ U(-1,1); w ~ N(0, 1/fan_in); b0 ~ N(0, 1/D); b1U ~ N(0, 1/H); b1q = 0.
    Values are rounded to float32 so that the oracle (fp64 arithmetic) and the
    GPU (fp32 arithmetic) see the SAME parameter values.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    T, H, D = model.n_types, model.n_neurons, model.n_desc
    nr = T * T * (model.n_max_r + 1) * (model.basis_r + 1)
    na = T * T * (model.n_max_a + 1) * (model.basis_a + 1)
    parts = [rng.uniform(-1.0, 1.0, nr), rng.uniform(-1.0, 1.0, na)]
    parts.append(np.ones(D) if scaler is None else np.asarray(scaler, dtype=np.float64))
    for _ in range(T):
        parts.append(rng.normal(0.0, 1.0 / np.sqrt(D), H * D))   # w0[H][D]
        parts.append(rng.normal(0.0, 1.0 / np.sqrt(D), H))       # b0[H]
        parts.append(rng.normal(0.0, 1.0 / np.sqrt(H), H))       # w1U[H]
        parts.append(rng.normal(0.0, 1.0 / np.sqrt(H), H))       # w1q[H]
    parts.append(rng.normal(0.0, 1.0 / np.sqrt(H), 1))           # b1U
    parts.append(np.zeros(1))                                    # b1q
    p = np.concatenate(parts).astype(np.float32)
    assert p.shape[0] == model.n_params()
    return p


def param_offsets(model: ModelDesc) -> dict:
    """Offsets of each block inside the flat parameter vector."""
    T, H, D = model.n_types, model.n_neurons, model.n_desc
    nr = T * T * (model.n_max_r + 1) * (model.basis_r + 1)
    na = T * T * (model.n_max_a + 1) * (model.basis_a + 1)
    off = {"c_r": 0, "c_a": nr, "scaler": nr + na, "nn": nr + na + D}
    off["per_type"] = H * D + 3 * H
    off["b1"] = off["nn"] + T * off["per_type"]
    return off


# ----------------------------------------------------------------------------
# structures
# ----------------------------------------------------------------------------
def _cubic_box(L: float) -> np.ndarray:
    return np.array([L, 0, 0, 0, L, 0, 0, 0, L], dtype=np.float64)


def rocksalt_lattice(n: int = 4, spacing: float = 2.82):
    """n^3 simple-cubic sites, type = (i+j+k) mod 2 (rock-salt ordering)."""
    g = np.arange(n)
    i, j, k = np.meshgrid(g, g, g, indexing="ij")
    pos = np.stack([i.ravel(), j.ravel(), k.ravel()]).astype(np.float64) * spacing
    types = ((i + j + k) % 2).ravel().astype(np.int32)
    return pos, types, _cubic_box(n * spacing)


def _random_rotations(rng, m):
    """m uniformly random rotation matrices (normalised Gaussian quaternions)."""
    q = rng.normal(size=(m, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    R = np.empty((m, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z)
    R[:, 0, 1] = 2 * (x * y - z * w)
    R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w)
    R[:, 1, 1] = 1 - 2 * (x * x + z * z)
    R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w)
    R[:, 2, 1] = 2 * (y * z + x * w)
    R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def water_box(n_side: int, seed: int, spacing: float = 3.104, jitter: float = 0.25,
              r_oh: float = 0.96, angle_deg: float = 104.5, d_min: float = 0.8):
    """n_side^3 rigid H2O on a jittered grid with random orientations.

    Atom order: O, H, H per molecule; types O = 0, H = 1.  A molecule's
    rotation is re-drawn while any intermolecular distance is < d_min.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    m = n_side ** 3
    L = n_side * spacing
    g = np.arange(n_side)
    i, j, k = np.meshgrid(g, g, g, indexing="ij")
    centres = (np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1) + 0.5) * spacing
    centres = centres + rng.uniform(-jitter, jitter, size=(m, 3))
    half = np.deg2rad(angle_deg) / 2
    local = np.array([[0.0, 0.0, 0.0],
                      [r_oh * np.sin(half), 0.0, r_oh * np.cos(half)],
                      [-r_oh * np.sin(half), 0.0, r_oh * np.cos(half)]])
    R = _random_rotations(rng, m)
    mol = np.repeat(np.arange(m), 3)
    for _ in range(200):
        xyz = centres[:, None, :] + np.einsum("mab,kb->mka", R, local)
        flat = np.mod(xyz.reshape(-1, 3), L)
        tree = cKDTree(flat, boxsize=L)
        pairs = tree.query_pairs(d_min, output_type="ndarray")
        if pairs.shape[0]:
            pairs = pairs[mol[pairs[:, 0]] != mol[pairs[:, 1]]]
        if pairs.shape[0] == 0:
            break
        bad = np.unique(mol[pairs[:, 1]])
        R[bad] = _random_rotations(rng, bad.shape[0])
    else:
        raise RuntimeError("water_box: could not remove close contacts")
    pos = np.ascontiguousarray(flat.T)
    types = np.tile(np.array([0, 1, 1], dtype=np.int32), m)
    return pos, types, _cubic_box(L)


def garnet_like(seed: int, n_grid: int = 30, spacing: float = 2.23, n_fu: int = 1088,
                sigma: float = 0.15, d_min: float = 1.6):
    """Li7La3Zr2O12-like stoichiometric random fill of a simple-cubic site grid (S14).

    types: Li = 0, La = 1, Zr = 2, O = 3.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    counts = np.array([7, 3, 2, 12]) * n_fu
    n = int(counts.sum())
    L = n_grid * spacing
    sites = rng.permutation(n_grid ** 3)[:n]
    ijk = np.stack(np.unravel_index(sites, (n_grid,) * 3), axis=1).astype(np.float64)
    base = (ijk + 0.5) * spacing
    types = rng.permutation(np.repeat(np.arange(4, dtype=np.int32), counts))
    disp = rng.normal(0.0, sigma, size=(n, 3))
    for _ in range(200):
        xyz = np.mod(base + disp, L)
        pairs = cKDTree(xyz, boxsize=L).query_pairs(d_min, output_type="ndarray")
        if pairs.shape[0] == 0:
            break
        bad = np.unique(pairs[:, 1])
        disp[bad] = rng.normal(0.0, sigma, size=(bad.shape[0], 3))
    else:
        raise RuntimeError("garnet_like: could not enforce the minimum separation")
    return np.ascontiguousarray(xyz.T), types, _cubic_box(L)


def perovskite(n_cells: int, seed: int, a: float = 4.0, sigma: float = 0.08):
    """BaTiO3-like cubic perovskite: Ba corner (0), Ti body centre (1), O faces (2)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    g = np.arange(n_cells)
    i, j, k = np.meshgrid(g, g, g, indexing="ij")
    cells = np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1).astype(np.float64)
    basis = np.array([[0, 0, 0], [.5, .5, .5], [.5, .5, 0], [.5, 0, .5], [0, .5, .5]])
    btypes = np.array([0, 1, 2, 2, 2], dtype=np.int32)
    xyz = (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a
    types = np.tile(btypes, cells.shape[0])
    L = n_cells * a
    xyz = np.mod(xyz + rng.normal(0.0, sigma, size=xyz.shape), L)
    return np.ascontiguousarray(xyz.T), types, _cubic_box(L)


# ----------------------------------------------------------------------------
# the BASELINE.json configs
# ----------------------------------------------------------------------------
MASSES_WATER = np.array([15.999, 1.008])


def config0(mode: int = 2, perturb: bool = True) -> Workload:
    """Tiny qNEP+Ewald: 64 atoms, 2 species, L = 11.28 A (BASELINE.json configs[0])."""
    seed = BASE_SEED + 0
    pos, types, box = rocksalt_lattice(4, 2.82)
    if perturb:
        rng = np.random.Generator(np.random.PCG64(seed))
        pos = np.mod(pos + rng.normal(0.0, 0.1, size=pos.shape), box[0])
    model = ModelDesc(n_types=2, n_neurons=30, mode=mode)
    params = random_params(model, seed + 1000, load_scaler("config0", model.n_desc))
    es = EsDesc(method=1, alpha=0.3, ewald_nmax2=64)
    return Workload("config0_tiny_ewald", pos, types, box, model, params, es)


def water_workload(n_side: int, grid: int, seed: int, name: str, mode: int = 2, key: str = "config1") -> Workload:
    pos, types, box = water_box(n_side, seed)
    model = ModelDesc(n_types=2, n_neurons=80, mode=mode)
    params = random_params(model, BASE_SEED + int(key[-1]) + 1000, load_scaler(key, model.n_desc))
    es = EsDesc(method=2, alpha=0.3, grid=(grid,) * 3, order=5)
    return Workload(name, pos, types, box, model, params, es, masses=MASSES_WATER.copy())


def config1(mode: int = 2) -> Workload:
    """Water-like box, 3000 atoms, PPPM 32^3 (BASELINE.json configs[1])."""
    return water_workload(10, 32, BASE_SEED + 1, "config1_water3k_pppm32", mode)


def config2(mode: int = 2) -> Workload:
    """Garnet-like 26112 atoms, 4 species, PPPM 64^3 (BASELINE.json configs[2], S14)."""
    seed = BASE_SEED + 2
    pos, types, box = garnet_like(seed)
    model = ModelDesc(n_types=4, n_neurons=80, mode=mode)
    params = random_params(model, seed + 1000, load_scaler("config2", model.n_desc))
    es = EsDesc(method=2, alpha=0.3, grid=(64,) * 3, order=5)
    return Workload("config2_garnet26k_pppm64", pos, types, box, model, params, es)


def config3(mode: int = 2, n_cells: int = 40, grid: int = 128, method: int = 2) -> Workload:
    """BaTiO3-like 40^3 cells = 320000 atoms, PPPM 128^3 (BASELINE.json configs[3]).

    ``n_cells=8, grid=32`` with ``method`` 1 or 2 gives the 2560-atom Ewald/PPPM cross-check.
    """
    seed = BASE_SEED + 3
    pos, types, box = perovskite(n_cells, seed)
    model = ModelDesc(n_types=3, n_neurons=80, mode=mode)
    params = random_params(model, seed + 1000, load_scaler("config3", model.n_desc))
    es = EsDesc(method=method, alpha=0.3, ewald_nmax2=64, grid=(grid,) * 3, order=5)
    return Workload(f"config3_perovskite{n_cells}_m{method}_g{grid}", pos, types, box, model, params, es)


def config4(mode: int = 2, n_side: int = 70, grid: int = 256) -> Workload:
    """Million-atom water-like box: 70^3 H2O = 1,029,000 atoms, PPPM 256^3 (configs[4])."""
    return water_workload(n_side, grid, BASE_SEED + 4, f"config4_water{3 * n_side ** 3}_pppm{grid}", mode,
                          key="config4")


def with_higher_body_terms(w: Workload, key: str) -> Workload:
    """The same structure with NEP4's 4- and 5-body angular terms switched on (10 more descriptors): new random parameters
    of the larger network (seed of the config + 5000), scaler from scalers.json[key]."""
    from dataclasses import replace
    m = replace(w.model, l_max_4b=2, l_max_5b=1)
    seed = BASE_SEED + 6000 + sum(ord(c) for c in key)
    return replace(w, model=m, params=random_params(m, seed, load_scaler(key, m.n_desc)), name=w.name + "_45body")


def triclinic_variant(w: Workload, tilt=((0.0, 0.0, 0.0), (0.18, 0.0, 0.0), (0.07, -0.12, 0.0))) -> Workload:
    """The same fractional coordinates in a tilted cell: row b gets tilt[b][a] * L_a added along a (lower-triangular
    tilts keep the cell volume).  Stands in for the non-orthogonal cells of PAPER.md :104."""
    from dataclasses import replace
    h = w.box.reshape(3, 3)
    hp = h + np.asarray(tilt, dtype=np.float64) @ np.diag(np.diag(h))
    frac = np.linalg.solve(h.T, w.pos)
    return replace(w, pos=np.ascontiguousarray(hp.T @ frac), box=hp.ravel().copy(), name=w.name + "_triclinic")


def maxwell_boltzmann(w: Workload, temperature: float = 300.0, seed: int | None = None) -> np.ndarray:
    """Velocities [3][N] in A / (natural time unit), natural unit = A*sqrt(amu/eV)."""
    kB = 8.617333262e-5  # eV/K
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 99 if seed is None else seed))
    m = w.masses[w.types]
    v = rng.normal(size=(3, w.n_atoms)) * np.sqrt(kB * temperature / m)[None, :]
    v -= (v * m).sum(axis=1, keepdims=True) / m.sum()
    return v


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}
