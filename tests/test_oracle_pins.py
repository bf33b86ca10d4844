"""Pins of the fp64 oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself through the same formula: each uses a closed form,
a library routine (numpy FFT, scipy spherical harmonics / B-splines / Chebyshev), brute force, a
finite difference of the oracle's own ENERGY / CHARGES, or an exact invariant.
"""
import os
from dataclasses import replace

import numpy as np
import pytest

import qnep_inputs as I

K = 14.3996454784
GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as _f:
    for _line in _f:
        if _line.strip() and not _line.startswith("#"):
            _k, _v = _line.split()[:2]
            GOLD[_k] = float(_v)


def rel_rms(a, b):
    return np.sqrt(((a - b) ** 2).sum() / (b ** 2).sum())


# ---------------------------------------------------------------- P1 Madelung
def test_madelung_converged(oracle):
    pos, types, box = I.rocksalt_lattice(4, 2.82)
    q = np.where(types == 0, 1.0, -1.0)
    es = I.EsDesc(method=1, alpha=0.6, ewald_nmax2=144)
    r = oracle.electrostatics(pos, q, box, 11.0, 1, es)
    M = -r["U"].sum() * 2.82 / (K * 32)
    assert abs(M - GOLD["madelung_nacl"]) < 2e-6
    # perfect lattice: every force vanishes, phi_i = -/+ M K / r0
    assert np.abs(r["F"]).max() < 1e-9
    assert np.allclose(r["phi"] * q, -GOLD["madelung_nacl"] * K / 2.82, rtol=2e-6)


def test_madelung_paper_defaults(oracle):
    """alpha = pi/r_c (:91) and kmax = 2 pi alpha (:110) give 'approximately 1e-5'."""
    pos, types, box = I.rocksalt_lattice(4, 2.82)
    q = np.where(types == 0, 1.0, -1.0)
    es = I.EsDesc(method=1, alpha=-1.0, ewald_nmax2=0)
    r = oracle.electrostatics(pos, q, box, 6.0, 1, es)
    M = -r["U"].sum() * 2.82 / (K * 32)
    err = abs(M - GOLD["madelung_nacl"])
    assert 1e-6 < err < 5 * GOLD["ewald_accuracy"]


# ------------------------------------------- P2 Ewald vs brute-force image sum
def _cubic_cluster(L):
    """Neutral cell with full cubic point symmetry: dipole and quadrupole vanish, so the
    shell-by-shell Coulomb sum converges fast and has no surface term."""
    a, b = 0.21 * L, 0.13 * L
    pts, q = [[0.0, 0.0, 0.0]], [-6.0 + 8 * 0.5]
    for ax in range(3):
        for s in (-1, 1):
            v = [0.0, 0.0, 0.0]
            v[ax] = s * a
            pts.append(v)
            q.append(1.0)
    for sx in (-1, 1):
        for sy in (-1, 1):
            for sz in (-1, 1):
                pts.append([sx * b, sy * b, sz * b])
                q.append(-0.5)
    pos = (np.array(pts) + L / 2).T.copy()
    q = np.array(q)
    assert abs(q.sum()) < 1e-14
    return pos, q


def test_ewald_vs_bruteforce_images(oracle):
    L = 7.0
    pos, q = _cubic_cluster(L)
    n = pos.shape[1]
    box = np.diag([L, L, L]).ravel()
    es = I.EsDesc(method=1, alpha=0.75, ewald_nmax2=196)
    r = oracle.electrostatics(pos, q, box, 13.9, 1, es)
    # brute force: sum over image cells in growing cubes
    M = 12
    g = np.arange(-M, M + 1)
    S = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3) * L
    d = pos.T[:, None, None, :] - pos.T[None, :, None, :] - S[None, None, :, :]   # r_i - r_j - s
    dist = np.linalg.norm(d, axis=-1)
    qq = q[:, None, None] * q[None, :, None]
    with np.errstate(divide="ignore", invalid="ignore"):
        inv = np.where(dist > 0, 1.0 / dist, 0.0)
        U = 0.5 * K * (qq * inv).sum()
        F = K * (qq[..., None] * d * inv[..., None] ** 3).sum(axis=(1, 2))
    assert abs(U - r["U"].sum()) < 1e-7 * abs(U)
    assert rel_rms(r["F"].T, F) < 1e-6
    assert np.abs(F).max() > 0.1     # the test is not vacuous


# ----------------------------------------------- P3 / P4 split consistency
def _random_charges(n, L, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    pos = rng.uniform(0, L, size=(3, n))
    q = rng.normal(size=n)
    q -= q.mean()
    return pos, q


def test_ewald_alpha_independence_and_phi_identity(oracle):
    L = 14.0
    pos, q = _random_charges(40, L, 7)
    box = np.diag([L, L, L]).ravel()
    res = []
    for alpha, nmax2 in ((0.55, 196), (0.75, 400)):
        r = oracle.electrostatics(pos, q, box, 13.5, 1, I.EsDesc(method=1, alpha=alpha, ewald_nmax2=nmax2))
        res.append(r)
        # P4: U^ES = 1/2 sum q_i phi_i (phi includes phi^s, and 1/2 sum q phi^s = U^s)
        assert abs(0.5 * (q * r["phi"]).sum() - r["U"].sum()) < 1e-10 * abs(r["U"].sum())
        # Eq. 10 closed form
        assert np.isclose(r["U"][2], -K * alpha / np.sqrt(np.pi) * (q ** 2).sum(), rtol=1e-13)
    a, b = res
    assert abs(a["U"].sum() - b["U"].sum()) < 1e-7 * abs(a["U"].sum())
    assert rel_rms(a["F"], b["F"]) < 1e-7
    assert np.abs(a["phi"] - b["phi"]).max() < 1e-6
    assert np.abs(a["W"] - b["W"]).max() < 1e-6 * np.abs(a["W"]).max()
    # the parts themselves differ (the test is not vacuous)
    assert abs(a["U"][1] - b["U"][1]) > 1e-2


def test_static_force_and_virial_are_derivatives_of_the_energy(oracle):
    """Eq. 15/18 = -dU/dr and Eq. 12/22 = -dU/d(strain) for fixed charges (mode 1, converged)."""
    L = 12.0
    pos, q = _random_charges(24, L, 11)
    box = np.diag([L, L, L]).ravel()
    es = I.EsDesc(method=1, alpha=0.8, ewald_nmax2=225)
    rc = 5.9      # alpha rc = 4.7: the truncation jump K erfc(4.7)/rc is ~1e-10 (S17)
    r0 = oracle.electrostatics(pos, q, box, rc, 1, es)
    h = 1e-5
    for (a, i) in ((0, 3), (1, 7), (2, 20)):
        p1, p2 = pos.copy(), pos.copy()
        p1[a, i] += h
        p2[a, i] -= h
        fd = -(oracle.electrostatics(p1, q, box, rc, 1, es)["U"].sum()
               - oracle.electrostatics(p2, q, box, rc, 1, es)["U"].sum()) / (2 * h)
        assert abs(fd - r0["F"][a, i]) < 2e-7 * max(1.0, abs(fd))
    # finite strain, integer k-set fixed (nmax2 criterion)
    for (a, b) in ((0, 0), (1, 2), (2, 1), (0, 1)):
        eps = np.zeros((3, 3))
        eps[a, b] = h
        def energy(sign):
            Fm = np.eye(3) + sign * eps
            return oracle.electrostatics(Fm @ pos, q, (box.reshape(3, 3) @ Fm.T).ravel(), rc, 1, es)["U"].sum()
        fd = -(energy(1) - energy(-1)) / (2 * h)
        assert abs(fd - r0["W"][a, b]) < 5e-7 * np.abs(r0["W"]).max()
    assert np.allclose(r0["W"], r0["W"].T, atol=1e-10)


# ------------------------------------------------------------- P12 FFT, W, d(z)
def test_fft_vs_numpy(oracle):
    rng = np.random.Generator(np.random.PCG64(3))
    x = rng.normal(size=(8, 4, 16)) + 1j * rng.normal(size=(8, 4, 16))
    assert np.allclose(oracle.fft3d(x, -1), np.fft.fftn(x), atol=1e-12)
    assert np.allclose(oracle.fft3d(x, +1), np.fft.ifftn(x) * x.size, atol=1e-12)


def test_bspline_vs_library_definition(oracle):
    from scipy.interpolate import BSpline
    b = BSpline.basis_element(np.arange(6) - 2.5)      # centred cardinal B-spline of order 5
    for dx in (-0.5, -0.31, 0.0, 0.123, 0.4999):
        w = oracle.bspline5(dx)
        ref = np.array([b(dx - o) if abs(dx - o) < 2.5 else 0.0 for o in (-2, -1, 0, 1, 2)])
        ref = np.nan_to_num(ref)
        assert np.allclose(w, ref, atol=1e-14), (dx, w, ref)
        assert abs(w.sum() - 1.0) < 1e-14


def test_alias_denominator_vs_brute_sum(oracle):
    """G2: d(z) = sum_m sinc^10(x + pi m), z = sin x -- fixes the sign of the 17/189 term."""
    m = np.arange(-4000, 4001)
    for x in (0.1, 0.7, 1.2, np.pi / 2):
        brute = (np.sinc((x + np.pi * m) / np.pi) ** 10).sum()
        assert abs(oracle.alias_denominator(np.sin(x)) - brute) < 1e-13


# --------------------------------------------------------------- P6 / P7 PPPM
def test_pppm_adjointness_identity(oracle):
    """U^k_mesh = 1/2 sum_i q_i phi^k_i exactly (Eq. 34 vs Eq. 38): pins the FFT normalisation (S11)
    and that spreading and back-interpolation use the same W."""
    L = 13.0
    pos, q = _random_charges(50, L, 5)
    box = np.diag([L, L, L]).ravel()
    r = oracle.electrostatics(pos, q, box, 6.0, 2, I.EsDesc(method=2, alpha=0.3, grid=(16, 16, 16)), want_rho=True)
    assert abs(0.5 * (q * r["phi"]).sum() - r["U"][1]) < 1e-12 * abs(r["U"][1])
    assert abs(r["rho"].sum() - q.sum()) < 1e-12          # W sums to one
    assert np.abs(r["F"].sum(axis=1)).max() < 1e-10         # P9: static mesh force sums to zero
    # phi^k is the exact charge-derivative of the mesh energy
    h = 1e-5
    for i in (0, 17):
        q1, q2 = q.copy(), q.copy()
        q1[i] += h
        q2[i] -= h
        es = I.EsDesc(method=2, alpha=0.3, grid=(16, 16, 16))
        fd = (oracle.electrostatics(pos, q1, box, 6.0, 2, es)["U"][1]
              - oracle.electrostatics(pos, q2, box, 6.0, 2, es)["U"][1]) / (2 * h)
        assert abs(fd - r["phi"][i]) < 1e-8


def test_pppm_converges_to_ewald(oracle):
    """P7 / G2: rel. force error falls as the mesh is refined and is ~1e-5..1e-4 at h ~ 1 A (:280)."""
    L = 16.0
    pos, q = _random_charges(120, L, 9)
    box = np.diag([L, L, L]).ravel()
    ew = oracle.electrostatics(pos, q, box, 6.0, 2, I.EsDesc(method=1, alpha=0.3, ewald_nmax2=169))
    errs = []
    for g in (16, 32, 64):
        pm = oracle.electrostatics(pos, q, box, 6.0, 2, I.EsDesc(method=2, alpha=0.3, grid=(g, g, g)))
        errs.append((rel_rms(pm["F"], ew["F"]), abs(pm["U"][1] - ew["U"][1]) / abs(ew["U"][1]),
                     rel_rms(pm["phi"], ew["phi"]), np.abs(pm["W"] - ew["W"]).max() / np.abs(ew["W"]).max()))
    assert errs[0][0] < GOLD["pppm_accuracy"] and errs[0][1] < 2e-5 and errs[0][2] < 1e-4 and errs[0][3] < 1e-4
    assert errs[1][0] < 3e-6 and errs[2][0] < 1e-7
    assert errs[2][1] < 1e-8 and errs[2][2] < 1e-7


# ------------------------------------------------ neighbours (a1): closed form + bins
def test_neighbor_counts_on_lattice(oracle):
    pos, types, box = I.rocksalt_lattice(4, 2.82)
    for rc in (4.0, 6.0):
        counts, _, _ = oracle.neighbors(pos, box, rc)
        g = np.arange(-4, 5)
        v = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
        d2 = (v ** 2).sum(1) * 2.82 ** 2
        expect = int(((d2 > 0) & (d2 < rc * rc)).sum())
        assert (counts == expect).all()


def test_binned_neighbors_equal_brute_force(oracle):
    rng = np.random.Generator(np.random.PCG64(17))
    box = np.array([13.0, 0, 0, 1.5, 14.0, 0, -1.0, 2.0, 15.0])     # triclinic
    pos = rng.uniform(-5, 20, size=(3, 400))
    rc = 4.0
    c0, j0, d0 = oracle.neighbors(pos, box, rc, use_bins=False, cap=96)
    c1, j1, d1 = oracle.neighbors(pos, box, rc, use_bins=True, cap=96)
    assert (c0 == c1).all() and c0.max() <= 96 and c0.min() > 0
    for i in range(400):
        a = sorted(zip(j0[i, :c0[i]], np.round(d0[i, :c0[i], 3], 9)))
        b = sorted(zip(j1[i, :c1[i]], np.round(d1[i, :c1[i], 3], 9)))
        assert a == b


# --------------------------------------------------- P10 descriptors vs library Y_lm
def test_descriptors_vs_spherical_harmonics(oracle):
    """Independent route (S1): D_nl = 4 pi/(2l+1) sum_m |sum_j g_n(r_ij) Y_lm(rhat_ij)|^2 with scipy's
    Y_lm and numpy's Chebyshev series -- the addition theorem must reproduce the Legendre double sum."""
    from numpy.polynomial import chebyshev as Ch
    try:
        from scipy.special import sph_harm_y
        Y = lambda l, m, theta, phi: sph_harm_y(l, m, theta, phi)
    except ImportError:       # older scipy
        from scipy.special import sph_harm
        Y = lambda l, m, theta, phi: sph_harm(m, l, phi, theta)
    w = I.config0()
    m = w.model
    p = w.params.astype(np.float64)
    off = I.param_offsets(m)
    nR, nA, Kb = m.n_max_r + 1, m.n_max_a + 1, m.basis_r + 1
    cR = p[off["c_r"]:off["c_a"]].reshape(2, 2, nR, Kb)
    cA = p[off["c_a"]:off["scaler"]].reshape(2, 2, nA, Kb)
    D = oracle.descriptors(m, p, w.pos, w.types, w.box)
    counts, jj, dd = oracle.neighbors(w.pos, w.box, m.rc_r, cap=48)

    def g(c, r, rc):
        x = 2 * (r / rc - 1) ** 2 - 1
        fc = 0.5 * (1 + np.cos(np.pi * r / rc))
        # sum_k c_k 1/2 (T_k(x) + 1) f_c
        return 0.5 * (Ch.chebval(x, c) + c.sum()) * fc

    for i in (0, 13, 40):
        ti = w.types[i]
        nb = [(jj[i, s], dd[i, s]) for s in range(counts[i])]
        Dn = np.zeros(m.n_desc)
        for n in range(nR):
            Dn[n] = sum(g(cR[ti, w.types[j], n], d[3], m.rc_r) for j, d in nb)
        ang = [(j, d) for j, d in nb if d[3] < m.rc_a]
        for n in range(nA):
            for l in range(1, m.l_max + 1):
                tot = 0.0
                for mm in range(-l, l + 1):
                    A = 0.0
                    for j, d in ang:
                        theta = np.arccos(d[2] / d[3])
                        phi = np.arctan2(d[1], d[0])
                        A += g(cA[ti, w.types[j], n], d[3], m.rc_a) * Y(l, mm, theta, phi)
                    tot += abs(A) ** 2
                Dn[nR + n * m.l_max + (l - 1)] = 4 * np.pi / (2 * l + 1) * tot
        assert np.allclose(D[i], Dn, rtol=1e-10, atol=1e-12)


# --------------------------------------------------- P5 / P8 full model derivatives
def _small_workload(mode, alpha):
    w = I.config0(mode=mode)
    w.es = replace(w.es, alpha=alpha, ewald_nmax2=36 if alpha < 0.5 else 300)
    return w


@pytest.mark.parametrize("mode,alpha", [(2, 0.3), (1, 0.8)])
def test_forces_are_minus_energy_gradient(oracle, mode, alpha):
    """Eq. 11, 14-19, 23 with the folding (:140) and S6: F = -dE/dr by central differences.
    Mode 1 uses alpha r_c = 4.8 so the real-space cutoff jump is negligible (S17)."""
    w = _small_workload(mode, alpha)
    out = oracle.compute_workload(w, use_bins=False)
    h = 1e-5
    for (a, i) in ((0, 0), (1, 21), (2, 63)):
        p1, p2 = w.pos.copy(), w.pos.copy()
        p1[a, i] += h
        p2[a, i] -= h
        e1 = oracle.compute(w.model, w.params, w.es, p1, w.types, w.box, use_bins=False)["energy"]
        e2 = oracle.compute(w.model, w.params, w.es, p2, w.types, w.box, use_bins=False)["energy"]
        fd = -(e1 - e2) / (2 * h)
        assert abs(fd - out["forces"][a, i]) < 2e-7 * max(1.0, abs(fd)), (fd, out["forces"][a, i])
    assert np.abs(out["forces"]).max() > 0.05
    assert np.abs(out["forces"].sum(axis=1)).max() < 1e-10          # P9
    assert abs(out["charges"].sum() - w.model.q_total) < 1e-12      # P9, Eq. 33 (G3)
    assert abs(out["energy_parts"]["k"]) > 1e-3                     # the charge path is exercised


@pytest.mark.parametrize("mode,alpha", [(2, 0.3), (1, 0.8)])
def test_virial_is_minus_strain_derivative(oracle, mode, alpha):
    """Eq. 12 + Eq. 21-22: W = -dE/d(eps) under r -> (1+eps) r, cell -> (1+eps) cell, k-set fixed in integers."""
    w = _small_workload(mode, alpha)
    out = oracle.compute_workload(w, use_bins=False)
    h = 1e-5
    for (a, b) in ((0, 0), (2, 2), (0, 1), (2, 1)):
        eps = np.zeros((3, 3))
        eps[a, b] = h
        def energy(sign):
            Fm = np.eye(3) + sign * eps
            return oracle.compute(w.model, w.params, w.es, Fm @ w.pos, w.types,
                                  (w.box.reshape(3, 3) @ Fm.T).ravel(), use_bins=False)["energy"]
        fd = -(energy(1) - energy(-1)) / (2 * h)
        assert abs(fd - out["virial"][a, b]) < 1e-6 * np.abs(out["virial"]).max(), (fd, out["virial"][a, b])
    assert np.allclose(out["virial"], out["virial"].T, atol=1e-9 * np.abs(out["virial"]).max())


def test_translation_and_permutation_invariance(oracle):
    w = I.config0(mode=1)
    a = oracle.compute_workload(w, use_bins=False, want_bec=True)
    shift = np.array([[0.3712], [-5.17], [13.09]])
    b = oracle.compute(w.model, w.params, w.es, w.pos + shift, w.types, w.box, use_bins=False, want_bec=True)
    assert abs(a["energy"] - b["energy"]) < 1e-10
    assert np.abs(a["forces"] - b["forces"]).max() < 1e-10
    assert np.abs(a["charges"] - b["charges"]).max() < 1e-12
    assert np.abs(a["bec"] - b["bec"]).max() < 1e-10
    perm = np.random.Generator(np.random.PCG64(1)).permutation(w.n_atoms)
    c = oracle.compute(w.model, w.params, w.es, w.pos[:, perm], w.types[perm], w.box, use_bins=False)
    assert abs(a["energy"] - c["energy"]) < 1e-10
    assert np.abs(a["forces"][:, perm] - c["forces"]).max() < 1e-10


# ------------------------------------------------------------- P13 limits
def test_static_charge_limits(oracle):
    w = I.config0(mode=1)
    off = I.param_offsets(w.model)
    H, D = w.model.n_neurons, w.model.n_desc
    # (a) w1q = 0 -> uniform charges -> neutralised to zero -> pure NEP
    p = w.params.copy()
    for t in range(2):
        base = off["nn"] + t * off["per_type"] + H * D + 2 * H
        p[base:base + H] = 0.0
    a = oracle.compute(w.model, p, w.es, w.pos, w.types, w.box, use_bins=False)
    assert np.abs(a["charges"]).max() < 1e-15
    assert a["energy"] == a["energy_parts"]["nep"]
    # (b) w0 = 0 -> charges depend on the species only -> textbook fixed-charge Ewald forces
    p = w.params.copy()
    for t in range(2):
        base = off["nn"] + t * off["per_type"]
        p[base:base + H * D] = 0.0
    b = oracle.compute(w.model, p, w.es, w.pos, w.types, w.box, use_bins=False)
    q = b["charges"]
    assert np.ptp(q[w.types == 0]) < 1e-14 and abs(q[w.types == 0][0] + q[w.types == 1][0]) < 1e-14
    assert abs(q[0]) > 1e-3
    s = oracle.electrostatics(w.pos, q, w.box, w.model.rc_r, 1, w.es)
    assert np.abs(b["forces"] - s["F"]).max() < 1e-12
    assert np.abs(b["virial"] - s["W"]).max() < 1e-11
    assert abs(b["energy"] - b["energy_parts"]["nep"] - s["U"].sum()) < 1e-11


# ------------------------------------------------------------- P11 BEC
def test_bec_sum_rule_and_finite_difference_assembly(oracle):
    """Eq. 28 (S12): sum_i Z_i = Q I, and Z assembled in python from FINITE-DIFFERENCED dq_i/dr_j."""
    pos, types, box = I.rocksalt_lattice(3, 2.82)
    rng = np.random.Generator(np.random.PCG64(23))
    L = 14.0                                   # > 2 r_c: every (i, j) pair is seen through one image only
    pos = pos * (L / box[0]) * 0.55 + rng.normal(0, 0.1, pos.shape) + 1.0
    types = types.copy()
    box = np.diag([L, L, L]).ravel()
    model = I.ModelDesc(n_types=2, n_neurons=10, mode=2)
    params = I.random_params(model, 5)
    es = I.EsDesc(method=0)
    n = pos.shape[1]
    out = oracle.compute(model, params, es, pos, types, box, use_bins=False, want_bec=True, debug=True)
    Z = out["bec"].reshape(3, 3, n)
    qt = model.sqrt_eps_inf * out["charges"]
    assert np.abs(Z.sum(axis=2) - qt.sum() * np.eye(3)).max() < 1e-12
    # c[i][j][beta] = sqrt(eps) d q_i^raw / d r_j,beta  (j != i)
    h = 1e-5
    c = np.zeros((n, n, 3))
    for j in range(n):
        for b in range(3):
            p1, p2 = pos.copy(), pos.copy()
            p1[b, j] += h
            p2[b, j] -= h
            q1 = oracle.compute(model, params, es, p1, types, box, use_bins=False, debug=True)["q_raw"]
            q2 = oracle.compute(model, params, es, p2, types, box, use_bins=False, debug=True)["q_raw"]
            c[:, j, b] = model.sqrt_eps_inf * (q1 - q2) / (2 * h)
    _, jj, dd = oracle.neighbors(pos, box, model.rc_r, cap=n)
    Zfd = np.zeros((3, 3, n))
    for i in range(n):
        Zfd[:, :, i] += qt[i] * np.eye(3)
        for j in range(n):
            if j == i:
                continue
            rij = pos[:, j] - pos[:, i]
            rij -= L * np.round(rij / L)
            if np.linalg.norm(rij) >= model.rc_r:
                continue
            Zfd[:, :, i] += 0.5 * (np.outer(rij, c[i, j]) - np.outer(-rij, c[j, i]))
    assert np.abs(Z - Zfd).max() < 5e-8
    assert np.abs(Z - qt[None, None, :] * np.eye(3)[:, :, None]).max() > 1e-3


# ------------------------------------------------------------- Eq. 29-30: field response
def test_field_response_point_charge_limit_and_power_identity(oracle):
    """Pins for orc_response (PAPER.md :229-237).
    (a) Point-charge limit: with the descriptor scaler set to zero the network sees x = 0, the charges depend on the
        species only and the BEC is q~_i I, so Eq. 29 must give the textbook force q~_i E and Eq. 30 the textbook
        current sum_i q~_i v_i.
    (b) Power identity for position-dependent charges (Z_i not symmetric): sum_i F_i^ext . v_i = E . Pdot -- fails if
        the two equations contract DIFFERENT indices of Z (it is blind to transposing Z in both at once; that case is
        pinned by test_field_response_vs_polarization_finite_differences).
    (c) Acoustic sum rule: sum_i F_i^ext = (sum_i Z_i)^T E = Q~ E = 0 and a rigid translation carries no current."""
    w = I.config0(mode=2)
    rng = np.random.Generator(np.random.PCG64(77))
    n = w.n_atoms
    E = np.array([0.3, -0.7, 0.45])
    vel = rng.normal(0, 0.05, (3, n))
    # (a)
    m = w.model
    params = w.params.copy()
    nco = 2 * m.n_types ** 2 * (m.n_max_r + 1) * (m.basis_r + 1)
    D = (m.n_max_r + 1) + (m.n_max_a + 1) * m.l_max
    params[nco:nco + D] = 0.0                                     # scaler s = 0
    out = oracle.compute(m, params, I.EsDesc(method=0), w.pos, w.types, w.box, use_bins=False, want_bec=True)
    qt = m.sqrt_eps_inf * out["charges"]
    assert np.abs(qt).max() > 1e-3 and len(np.unique(np.round(qt, 12))) == m.n_types
    fext, pdot = oracle.response(out["bec"], E, vel)
    assert np.abs(fext - E[:, None] * qt[None, :]).max() < 1e-13
    assert np.abs(pdot - (vel * qt[None, :]).sum(axis=1)).max() < 1e-12
    # (b), (c)
    out = oracle.compute(m, w.params, I.EsDesc(method=0), w.pos, w.types, w.box, use_bins=False, want_bec=True)
    Z = out["bec"].reshape(3, 3, n)
    assert np.abs(Z - np.transpose(Z, (1, 0, 2))).max() > 1e-3    # the test is blind to transposition otherwise
    fext, pdot = oracle.response(out["bec"], E, vel)
    assert abs((fext * vel).sum() - E @ pdot) < 1e-12 * max(1.0, abs(E @ pdot))
    assert np.abs(fext.sum(axis=1)).max() < 1e-12
    _, p_rigid = oracle.response(out["bec"], None, np.repeat(np.array([[0.1], [0.2], [-0.3]]), n, axis=1))
    assert np.abs(p_rigid).max() < 1e-12
    # only one of the two outputs requested
    f_only, none = oracle.response(out["bec"], E, None)
    assert none is None and np.array_equal(f_only, fext)


# ------------------------------------------------------------- Eq. 1: hand-evaluated network
def _pin_model(H=2):
    m = I.ModelDesc(n_types=2, n_neurons=H, mode=2)
    p = np.zeros(m.n_params())
    off = I.param_offsets(m)
    return m, p, off


def test_nn_forward_hand_evaluated(oracle):
    """Eq. 1 (PAPER.md :41-45) and the charge node (:58-60) with every number typed by hand: pins the MINUS signs of
    b0 and b1 and the per-type weight blocks (S4).
    (a) scaler = 0: the network sees x = 0, so h = tanh(-b0).
        type 0: b0 = (-atanh 1/2, +atanh 1/4) -> h = (1/2, -1/4); w1U = (3, 8), w1q = (4, 4); b1U = 3/4, b1q = 1/8
                -> U = 3/2 - 2 - 3/4 = -5/4,  q = 2 - 1 - 1/8 = 7/8;
        type 1: b0 = (+atanh 1/2, 0) -> h = (-1/2, 0); w1U = (2, 5), w1q = (-2, 7)
                -> U = -1 - 3/4 = -7/4,  q = 1 - 1/8 = 7/8.
    (b) an isolated pair at r = r_c^R / 2 with c^R_{n k} = 2 delta_{n0} delta_{k0}, c^A = 0: f_0 = f_c = 1/2[1 + cos(pi/2)]
        = 1/2, so D_0 = 1 exactly and all other descriptors vanish.  With s_0 = 1, w0[mu][0] = (2 atanh 1/2, 0),
        b0 = (atanh 1/2, -atanh 1/4): z = (atanh 1/2, atanh 1/4), h = (1/2, 1/4) -> the w0 . D term enters with PLUS,
        the bias with MINUS (with +b0, h_0 would be tanh(3 atanh 1/2) = 13/14)."""
    a2, a4 = np.arctanh(0.5), np.arctanh(0.25)
    # ---- (a)
    m, p, off = _pin_model()
    H, D = 2, m.n_desc
    t0, t1 = off["nn"], off["nn"] + off["per_type"]
    p[t0 + H * D: t0 + H * D + 2] = [-a2, a4]          # b0, type 0
    p[t0 + H * D + 2: t0 + H * D + 4] = [3.0, 8.0]     # w1U
    p[t0 + H * D + 4: t0 + H * D + 6] = [4.0, 4.0]     # w1q
    p[t1 + H * D: t1 + H * D + 2] = [a2, 0.0]          # b0, type 1
    p[t1 + H * D + 2: t1 + H * D + 4] = [2.0, 5.0]
    p[t1 + H * D + 4: t1 + H * D + 6] = [-2.0, 7.0]
    p[off["b1"]], p[off["b1"] + 1] = 0.75, 0.125
    p[off["c_r"]:off["scaler"]] = 0.37                 # descriptors are non-zero but the scaler (= 0) hides them
    w = I.config0(mode=2)
    out = oracle.compute(m, p, I.EsDesc(method=0), w.pos, w.types, w.box, use_bins=False, debug=True)
    assert np.abs(out["D"]).max() > 0.1
    U0, q0, U1, q1 = -1.25, 0.875, -1.75, 0.875         # typed from Eq. 1, see the docstring
    assert np.abs(out["U_i"][w.types == 0] - U0).max() < 1e-14
    assert np.abs(out["q_raw"][w.types == 0] - q0).max() < 1e-14
    assert np.abs(out["U_i"][w.types == 1] - U1).max() < 1e-14
    assert np.abs(out["q_raw"][w.types == 1] - q1).max() < 1e-14
    assert abs(out["energy"] - (32 * U0 + 32 * U1)) < 1e-12                      # Eq. 2
    # ---- (b)
    m, p, off = _pin_model()
    nb = m.basis_r + 1
    nR = m.n_max_r + 1
    for ti in range(2):
        for tj in range(2):
            p[off["c_r"] + ((ti * 2 + tj) * nR + 0) * nb + 0] = 2.0
    p[off["scaler"]] = 1.0
    for t in (0, 1):
        b = off["nn"] + t * off["per_type"]
        p[b + 0 * D + 0] = 2.0 * a2                     # w0[0][0]
        p[b + H * D: b + H * D + 2] = [a2, -a4]         # b0
        p[b + H * D + 2: b + H * D + 4] = [4.0, 8.0]    # w1U
        p[b + H * D + 4: b + H * D + 6] = [2.0, -4.0]   # w1q
    p[off["b1"]], p[off["b1"] + 1] = -0.5, 0.25
    L = 40.0
    pos = np.array([[10.0, 10.0 + 3.0 / np.sqrt(3)], [12.0, 12.0 + 3.0 / np.sqrt(3)], [9.0, 9.0 + 3.0 / np.sqrt(3)]])
    out = oracle.compute(m, p, I.EsDesc(method=0), pos, np.array([0, 1], dtype=np.int32),
                         np.diag([L, L, L]).ravel(), use_bins=False, debug=True)
    expect_D = np.zeros(m.n_desc)
    expect_D[0] = 1.0
    assert np.abs(out["D"] - expect_D[None, :]).max() < 1e-14
    # h = (1/2, 1/4): U = 4/2 + 8/4 - (-1/2) = 9/2, q = 2/2 - 4/4 - 1/4 = -1/4
    assert np.abs(out["U_i"] - 4.5).max() < 1e-13
    assert np.abs(out["q_raw"] + 0.25).max() < 1e-13


# ------------------------------------------------------------- Eq. 26-30: cluster polarization
def _cluster():
    rng = np.random.Generator(np.random.PCG64(101))
    m = I.ModelDesc(n_types=2, n_neurons=8, mode=2)
    p = I.random_params(m, 9).astype(np.float64)
    L = 40.0
    pos = (np.array([[0.0, 2.1, -0.4, 1.3, -1.9], [0.0, 0.3, 2.2, -1.7, -0.8], [0.0, -0.6, 0.9, 1.6, 2.0]])
           + rng.normal(0, 0.05, (3, 5)) + 20.0)
    types = np.array([0, 1, 1, 0, 1], dtype=np.int32)
    return m, p, pos, types, np.diag([L, L, L]).ravel()


def test_cluster_polarization_derivative_vs_bec(oracle):
    """P11, second half, and the index order of Z (PAPER.md :216-227, Eq. 26-28).
    For an isolated cluster P_a = sum_i q~_i r_ia (Eq. 26) is well defined and Z_{i,ab} = dP_a / dr_ib (Eq. 27).
    Finite differences of P (from the oracle's CHARGES only) are compared with the oracle's BEC output (Eq. 28):
      * dimer: Eq. 28 equals dP/dr exactly (r_i + r_j = 2 rbar);
      * general cluster: Eq. 28 is a different per-atom partition of the same total; with c_ij = d q~_i / d r_ij
        (finite differences of q_raw, S12)   Z^(28)_i,ab - dP_a/dr_ib = 1/2 sum_j (r_i + r_j - 2 rbar)_a (c_ij - c_ji)_b
        (rbar enters through the Eq. 33 shift, whose derivative Eq. 28 drops).  DESIGN.md reading S12b.
    Both are asymmetric in (a, b): a transposed BEC layout fails."""
    m, p, pos, types, box = _cluster()
    es = I.EsDesc(method=0)
    h = 1e-5

    def run(x, ty):
        return oracle.compute(m, p, es, x, ty, box, use_bins=False, want_bec=True, debug=True)

    def P(x, ty):
        return m.sqrt_eps_inf * (run(x, ty)["charges"][None, :] * x).sum(axis=1)

    def dP(x, ty):
        n = x.shape[1]
        Z = np.zeros((3, 3, n))
        for i in range(n):
            for b in range(3):
                x1, x2 = x.copy(), x.copy()
                x1[b, i] += h
                x2[b, i] -= h
                Z[:, b, i] = (P(x1, ty) - P(x2, ty)) / (2 * h)
        return Z

    # dimer
    xd, td = pos[:, :2].copy(), types[:2].copy()
    Zd = run(xd, td)["bec"].reshape(3, 3, 2)
    assert np.abs(Zd - dP(xd, td)).max() < 2e-9
    assert np.abs(Zd - m.sqrt_eps_inf * run(xd, td)["charges"][None, None, :] * np.eye(3)[:, :, None]).max() > 1e-3
    # five atoms
    n = pos.shape[1]
    Z28 = run(pos, types)["bec"].reshape(3, 3, n)
    Zfd = dP(pos, types)
    c = np.zeros((n, n, 3))                         # c[i][j][b] = sqrt(eps) d q_raw_i / d r_jb = c_ij (j != i)
    for j in range(n):
        for b in range(3):
            x1, x2 = pos.copy(), pos.copy()
            x1[b, j] += h
            x2[b, j] -= h
            c[:, j, b] = m.sqrt_eps_inf * (run(x1, types)["q_raw"] - run(x2, types)["q_raw"]) / (2 * h)
    rbar = pos.mean(axis=1)
    corr = np.zeros((3, 3, n))
    for i in range(n):
        for j in range(n):
            if j != i:
                corr[:, :, i] += 0.5 * np.outer(pos[:, i] + pos[:, j] - 2 * rbar, c[i, j] - c[j, i])
    assert np.abs(corr).max() > 1e-3 and np.abs(Zfd - np.transpose(Zfd, (1, 0, 2))).max() > 1e-3
    assert np.abs(Z28 - corr - Zfd).max() < 5e-9
    assert np.abs(np.transpose(Z28, (1, 0, 2)) - corr - Zfd).max() > 1e-3      # the transposed layout is rejected


def test_field_response_vs_polarization_finite_differences(oracle):
    """Eq. 29-30 (PAPER.md :229-237) as the chain rule they are: with Z_{i,ab} = dP_a/dr_ib (here taken by finite
    differences of the cluster polarization, asymmetric),  F^ext_ib = d(E.P)/dr_ib  and  Pdot_a = dP_a/dt along the
    velocities.  Transposing Z in BOTH equations (which the power identity cannot see) fails here.  Plus one case
    evaluated by hand."""
    # by hand: one ion, Z_ab = 3a + b + 1, E = (1, 0, 0) -> F_b = Z_0b; v = (0, 0, 1) -> Pdot_a = Z_a2
    Z1 = np.arange(1.0, 10.0).reshape(9, 1)
    f, pd = oracle.response(Z1, np.array([1.0, 0.0, 0.0]), np.array([[0.0], [0.0], [1.0]]))
    assert np.array_equal(f[:, 0], [1.0, 2.0, 3.0]) and np.array_equal(pd, [3.0, 6.0, 9.0])
    f, pd = oracle.response(Z1, np.array([0.0, 2.0, -1.0]), np.array([[1.0], [-1.0], [0.5]]))
    assert np.array_equal(f[:, 0], [2 * 4.0 - 7.0, 2 * 5.0 - 8.0, 2 * 6.0 - 9.0])
    assert np.array_equal(pd, [1.0 - 2.0 + 1.5, 4.0 - 5.0 + 3.0, 7.0 - 8.0 + 4.5])
    # cluster
    m, p, pos, types, box = _cluster()
    es = I.EsDesc(method=0)
    n = pos.shape[1]
    h = 1e-5

    def P(x):
        q = oracle.compute(m, p, es, x, types, box, use_bins=False)["charges"]
        return m.sqrt_eps_inf * (q[None, :] * x).sum(axis=1)

    Z = np.zeros((9, n))
    for i in range(n):
        for b in range(3):
            x1, x2 = pos.copy(), pos.copy()
            x1[b, i] += h
            x2[b, i] -= h
            Z[[b, 3 + b, 6 + b], i] = (P(x1) - P(x2)) / (2 * h)      # entry (3 a + b): dP_a / dr_ib
    rng = np.random.Generator(np.random.PCG64(5))
    E = np.array([0.4, -0.9, 0.25])
    vel = rng.normal(0, 1.0, (3, n))
    fext, pdot = oracle.response(Z, E, vel)
    dt = 1e-5
    pdot_fd = (P(pos + dt * vel) - P(pos - dt * vel)) / (2 * dt)
    assert np.abs(pdot - pdot_fd).max() < 1e-8 * max(1.0, np.abs(pdot_fd).max())
    fext_fd = np.zeros((3, n))
    for i in range(n):
        for b in range(3):
            x1, x2 = pos.copy(), pos.copy()
            x1[b, i] += h
            x2[b, i] -= h
            fext_fd[b, i] = (E @ P(x1) - E @ P(x2)) / (2 * h)
    assert np.abs(fext - fext_fd).max() < 1e-9
    Zt = Z.reshape(3, 3, n).transpose(1, 0, 2).reshape(9, n)
    ft, pt = oracle.response(Zt, E, vel)
    assert np.abs(ft - fext_fd).max() > 1e-3 and np.abs(pt - pdot_fd).max() > 1e-3


# ------------------------------------------------------------- per-atom virial (Eq. 12, 20, 39)
def test_atom_virial_static_coulomb_vs_bruteforce_and_trace(oracle):
    """Eq. 12 + Eq. 15 (real space) and Eq. 20 (reciprocal space, real part: reading G4) for FIXED charges, converged:
    (a) against the pairwise definition W_i = 1/2 sum_j sum_images K q_i q_j r (x) r / r^3 summed by brute force over
        image cubes of a neutral cell with cubic point symmetry (no dipole, isotropic second moment);
    (b) Tr W_i = 1/2 q_i phi_i for every atom (the Coulomb virial theorem per atom; phi includes the self term);
    (c) sum_i W_i = W (Eq. 22 + Eq. 12), W_i symmetric."""
    L = 7.0
    pos, q = _cubic_cluster(L)
    n = pos.shape[1]
    box = np.diag([L, L, L]).ravel()
    es = I.EsDesc(method=1, alpha=0.75, ewald_nmax2=196)
    r = oracle.electrostatics(pos, q, box, 13.9, 1, es, want_atom_virial=True)
    Wat = r["W_atom"].reshape(3, 3, n)
    M = 12
    g = np.arange(-M, M + 1)
    S = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3) * L
    d = pos.T[:, None, None, :] - pos.T[None, :, None, :] - S[None, None, :, :]
    dist = np.linalg.norm(d, axis=-1)
    qq = q[:, None, None] * q[None, :, None]
    with np.errstate(divide="ignore", invalid="ignore"):
        inv3 = np.where(dist > 0, 1.0 / dist ** 3, 0.0)
    brute = 0.5 * K * np.einsum("ijs,ijsa,ijsb->abi", qq * inv3, d, d)
    # Summed over cubes of images, the potential of a neutral cell without dipole still differs from the Ewald
    # (tin-foil) one by the constant c = -2 pi K / (3 V) sum_j q_j |r_j|^2 (the trace of the second moment); the
    # energy does not see it (sum q = 0), Tr W_i = 1/2 q_i phi_i does: W_i^brute = W_i^Ewald + (q_i c / 6) 1.
    c = -(2 * np.pi / (3 * L ** 3)) * K * (q * ((pos - L / 2) ** 2).sum(axis=0)).sum()
    shifted = brute - (q * c / 6.0)[None, None, :] * np.eye(3)[:, :, None]
    assert abs(c) > 0.1
    assert np.abs(Wat - shifted).max() < 1e-5 * np.abs(brute).max()
    assert np.abs(np.einsum("aai->i", Wat) - 0.5 * q * r["phi"]).max() < 1e-9 * np.abs(q * r["phi"]).max()
    assert np.abs(Wat.sum(axis=2) - r["W"]).max() < 1e-11 * np.abs(r["W"]).max()
    assert np.abs(Wat - np.transpose(Wat, (1, 0, 2))).max() < 1e-12
    assert np.abs(Wat[0, 1]).max() > 1e-3 * np.abs(Wat).max()          # off-diagonal elements are exercised


def test_atom_virial_pppm_converges_to_ewald_and_sums_to_total(oracle):
    """Eq. 39 (six inverse FFTs) against Eq. 20: same limit as the mesh is refined; sum_i W_i = W^k exactly (the
    adjointness of spreading and back-interpolation)."""
    L = 16.0
    pos, q = _random_charges(120, L, 9)
    box = np.diag([L, L, L]).ravel()
    ew = oracle.electrostatics(pos, q, box, 6.0, 2, I.EsDesc(method=1, alpha=0.3, ewald_nmax2=169), want_atom_virial=True)
    errs = []
    for g in (16, 32, 64):
        pm = oracle.electrostatics(pos, q, box, 6.0, 2, I.EsDesc(method=2, alpha=0.3, grid=(g, g, g)), want_atom_virial=True)
        assert np.abs(pm["W_atom"].reshape(3, 3, -1).sum(axis=2) - pm["W"]).max() < 1e-11 * np.abs(pm["W"]).max()
        errs.append(rel_rms(pm["W_atom"], ew["W_atom"]))
    assert errs[0] < 2e-4 and errs[1] < 1e-5 and errs[2] < 1e-6 and errs[2] < errs[1] < errs[0]


def test_atom_virial_pair_part_vs_site_energy_derivatives(oracle):
    """Eq. 12, W_i = sum_j r_ij (x) F_ji, with the partial force F_ji = dU_j / dr_ji = dU_j / dr_i (Eq. 14; the site
    energy of j depends on r_i only through r_ji): finite differences of the oracle's SITE ENERGIES fix which atom a
    pair term belongs to.  Cluster without electrostatics (the descriptor part of the path)."""
    m, p, pos, types, box = _cluster()
    n = pos.shape[1]
    es = I.EsDesc(method=0)
    out = oracle.compute(m, p, es, pos, types, box, use_bins=False, want_atom_virial=True)
    Wat = out["virial_atom"].reshape(3, 3, n)
    h = 1e-5
    ref = np.zeros((3, 3, n))
    for i in range(n):
        for b in range(3):
            x1, x2 = pos.copy(), pos.copy()
            x1[b, i] += h
            x2[b, i] -= h
            dU = (oracle.compute(m, p, es, x1, types, box, use_bins=False, debug=True)["U_i"]
                  - oracle.compute(m, p, es, x2, types, box, use_bins=False, debug=True)["U_i"]) / (2 * h)
            for j in range(n):
                if j != i:
                    ref[:, b, i] += (pos[:, j] - pos[:, i]) * dU[j]          # r_ij,a * dU_j/dr_i,b
    assert np.abs(Wat - ref).max() < 2e-8 * max(1.0, np.abs(ref).max())
    assert np.abs(Wat.sum(axis=2) - out["virial"]).max() < 1e-12 * max(1.0, np.abs(out["virial"]).max())
    # the partition differs from "every atom keeps its own -r_ij (x) F_ij": the test would see that assignment
    alt = np.zeros((3, 3, n))
    for j in range(n):
        for b in range(3):
            x1, x2 = pos.copy(), pos.copy()
            x1[b, j] += h
            x2[b, j] -= h
            dU = (oracle.compute(m, p, es, x1, types, box, use_bins=False, debug=True)["U_i"]
                  - oracle.compute(m, p, es, x2, types, box, use_bins=False, debug=True)["U_i"]) / (2 * h)
            for i in range(n):
                if i != j:
                    alt[:, b, i] += -(pos[:, j] - pos[:, i]) * dU[i]         # -r_ij,a * F_ij,b kept by atom i
    assert np.abs(alt - ref).max() > 1e-3


@pytest.mark.parametrize("mode,method", [(1, 1), (2, 1), (2, 2)])
def test_atom_virial_full_model_sums_to_total(oracle, mode, method):
    """All parts together (descriptor + dynamic-charge partial forces, Eq. 15 / 20 / 39 static parts)."""
    w = I.config0(mode=mode)
    if method == 2:
        w.es = replace(w.es, method=2, grid=(16, 16, 16))
    out = oracle.compute_workload(w, use_bins=False, want_atom_virial=True)
    Wat = out["virial_atom"].reshape(3, 3, -1)
    assert np.abs(Wat.sum(axis=2) - out["virial"]).max() < 1e-11 * np.abs(out["virial"]).max()
    assert np.abs(Wat).max() > 1e-2


# --------------------------------------------------- ZBL core (reading Z1)
def test_zbl_pair_limits_and_switch(oracle):
    """The screening function is normalised (phi(0) = 1), so U_ZBL -> K Z_i Z_j / r for r -> 0 (bare nuclei); the switch
    leaves the function untouched below r_1, takes it to zero with zero slope at r_2, and dU/dr is the derivative of U."""
    K = 14.3996454784
    for (Zi, Zj) in ((8.0, 1.0), (56.0, 22.0)):
        a = 0.46850 / (Zi ** 0.23 + Zj ** 0.23)
        for r in (1e-6, 1e-5):
            u, du = oracle.zbl_pair(r, Zi, Zj, 0.5, 1.0)
            # first-order screening correction: phi(x) = 1 - (sum_k c_k d_k) x + O(x^2)
            slope = 0.18175 * 3.19980 + 0.50986 * 0.94229 + 0.28022 * 0.40290 + 0.02817 * 0.20162
            assert abs(u * r / (K * Zi * Zj) - (1.0 - slope * r / a)) < 3.0 * (r / a) ** 2 + 1e-12      # O(x^2) remainder
        # below r_1 the switch is inactive: the value does not depend on (r_1, r_2)
        assert oracle.zbl_pair(0.4, Zi, Zj, 0.5, 1.0) == oracle.zbl_pair(0.4, Zi, Zj, 0.45, 3.0)
        # end of the switch: value and slope vanish, and nothing beyond
        u2, du2 = oracle.zbl_pair(1.0 - 1e-9, Zi, Zj, 0.5, 1.0)
        assert abs(u2) < 1e-12 * K * Zi * Zj and abs(du2) < 1e-6 * K * Zi * Zj
        assert oracle.zbl_pair(1.0, Zi, Zj, 0.5, 1.0) == (0.0, 0.0)
        # continuity of value and slope across r_1, and dU/dr against central differences inside the switch
        ua, dua = oracle.zbl_pair(0.5 - 1e-9, Zi, Zj, 0.5, 1.0)
        ub, dub = oracle.zbl_pair(0.5 + 1e-9, Zi, Zj, 0.5, 1.0)
        assert abs(ua - ub) < 1e-6 * abs(ua) and abs(dua - dub) < 1e-6 * abs(dua)
        for r in (0.3, 0.6, 0.9):
            h = 1e-6
            fd = (oracle.zbl_pair(r + h, Zi, Zj, 0.5, 1.0)[0] - oracle.zbl_pair(r - h, Zi, Zj, 0.5, 1.0)[0]) / (2 * h)
            assert abs(fd - oracle.zbl_pair(r, Zi, Zj, 0.5, 1.0)[1]) < 1e-7 * abs(fd)
        # repulsive and monotonically decreasing
        us = [oracle.zbl_pair(r, Zi, Zj, 0.5, 1.0)[0] for r in np.linspace(0.05, 0.99, 40)]
        assert all(x > y > 0 for x, y in zip(us, us[1:]))


def test_zbl_dimer_energy_is_the_pair_function(oracle):
    """Two atoms far from everything: the ZBL part of the energy is exactly U_ZBL(r) (1/2 per atom, one pair), the force is
    -U'(r) along the bond, and the term vanishes when the pair is beyond r_2."""
    w = I.config0(mode=2)
    w.es = replace(w.es, method=0)
    L = 40.0
    box = np.diag([L, L, L]).ravel()
    types = np.array([0, 1], dtype=np.int32)
    zbl = (1.0, 2.0, (11.0, 17.0))
    for r in (0.8, 1.5, 2.5):
        pos = np.array([[5.0, 5.0 + r * 0.6], [7.0, 7.0 + r * 0.8], [9.0, 9.0]])
        on = oracle.compute(w.model, w.params, w.es, pos, types, box, use_bins=False, zbl=zbl)
        off = oracle.compute(w.model, w.params, w.es, pos, types, box, use_bins=False)
        u, du = oracle.zbl_pair(r, 11.0, 17.0, 1.0, 2.0)
        assert abs(on["energy_parts"]["zbl"] - u) < 1e-12 * max(1.0, abs(u))
        assert abs((on["energy"] - off["energy"]) - u) < 1e-10 * max(1.0, abs(u))
        dF = on["forces"] - off["forces"]
        bond = np.array([0.6, 0.8, 0.0])
        assert np.allclose(dF[:, 1], -du * bond, atol=1e-10 * max(1.0, abs(du)))
        assert np.allclose(dF[:, 0], du * bond, atol=1e-10 * max(1.0, abs(du)))
        if r > 2.0:
            assert u == 0.0 and on["energy_parts"]["zbl"] == 0.0


def test_zbl_forces_and_virial_in_the_full_model(oracle):
    """With the ZBL term on (r_2 = 3.5 A on the 2.82 A lattice of config 0, so every nearest-neighbour pair is inside the
    switch), forces are still -dE/dr, the virial is -dE/d(strain), and the per-atom virial sums to the total."""
    w = _small_workload(2, 0.3)
    zbl = (1.5, 3.5, (11.0, 17.0))
    out = oracle.compute_workload(w, use_bins=False, zbl=zbl, want_atom_virial=True)
    base = oracle.compute_workload(w, use_bins=False)
    assert out["energy_parts"]["zbl"] > 1.0 and rel_rms(out["forces"], base["forces"]) > 1e-2
    h = 1e-5
    for (a, i) in ((0, 3), (2, 40)):
        p1, p2 = w.pos.copy(), w.pos.copy()
        p1[a, i] += h
        p2[a, i] -= h
        e1 = oracle.compute(w.model, w.params, w.es, p1, w.types, w.box, use_bins=False, zbl=zbl)["energy"]
        e2 = oracle.compute(w.model, w.params, w.es, p2, w.types, w.box, use_bins=False, zbl=zbl)["energy"]
        fd = -(e1 - e2) / (2 * h)
        assert abs(fd - out["forces"][a, i]) < 2e-7 * max(1.0, abs(fd)), (fd, out["forces"][a, i])
    for (a, b) in ((0, 0), (1, 2)):
        eps = np.zeros((3, 3))
        eps[a, b] = h
        def energy(sign):
            Fm = np.eye(3) + sign * eps
            return oracle.compute(w.model, w.params, w.es, Fm @ w.pos, w.types,
                                  (w.box.reshape(3, 3) @ Fm.T).ravel(), use_bins=False, zbl=zbl)["energy"]
        fd = -(energy(1) - energy(-1)) / (2 * h)
        assert abs(fd - out["virial"][a, b]) < 1e-6 * np.abs(out["virial"]).max(), (fd, out["virial"][a, b])
    assert np.abs(out["forces"].sum(axis=1)).max() < 1e-9
    assert np.allclose(out["virial_atom"].sum(axis=1).reshape(3, 3), out["virial"], atol=1e-9 * np.abs(out["virial"]).max())
    # the switch-off state leaks nowhere: a later call without zbl is the plain model again
    again = oracle.compute_workload(w, use_bins=False)
    assert abs(again["energy"] - base["energy"]) < 1e-12 and again["energy_parts"]["zbl"] == 0.0


# --------------------------------------------------- triclinic cells (PAPER.md :104)
def test_sheared_description_of_the_same_crystal(oracle):
    """A periodic crystal does not know which cell vectors describe it: the cubic box (a, b, c) and the sheared box
    (a + b, b, c + a) span the same lattice, so the whole model (neighbours over images, descriptors, network, Ewald with the
    |k| <= 2 pi alpha sphere of the paper, forces, virial, charges) must give the same numbers -- on a triclinic cell."""
    w = I.config0(mode=1)
    w.es = replace(w.es, alpha=0.6, ewald_nmax2=0)          # physical k sphere (:110): the same k set in both descriptions
    a = oracle.compute_workload(w, use_bins=False, want_bec=True, want_atom_virial=True)
    h = w.box.reshape(3, 3)
    sheared = np.array([h[0] + h[1], h[1], h[2] + h[0]])
    assert abs(np.linalg.det(sheared) - np.linalg.det(h)) < 1e-9
    for use_bins in (False, True):
        b = oracle.compute(w.model, w.params, w.es, w.pos, w.types, sheared.ravel(), use_bins=use_bins, want_bec=True,
                           want_atom_virial=True)
        assert abs(a["energy"] - b["energy"]) < 1e-9
        assert np.abs(a["forces"] - b["forces"]).max() < 1e-9
        assert np.abs(a["virial"] - b["virial"]).max() < 1e-8
        assert np.abs(a["charges"] - b["charges"]).max() < 1e-12
        assert np.abs(a["bec"] - b["bec"]).max() < 1e-9
        assert np.abs(a["virial_atom"] - b["virial_atom"]).max() < 1e-8


_triclinic = I.triclinic_variant


def test_triclinic_forces_and_virial_are_energy_derivatives(oracle):
    """Eq. 11-23 on a genuinely triclinic cell (Ewald): F = -dE/dr, W = -dE/d(strain), sum F = 0, W symmetric."""
    w = _triclinic(_small_workload(2, 0.3))
    hbox = w.box.reshape(3, 3)
    assert abs(hbox[1, 0]) > 1.0 and abs(hbox[2, 1]) > 1.0
    out = oracle.compute_workload(w, use_bins=False)
    h = 1e-5
    for (a, i) in ((0, 5), (1, 33), (2, 60)):
        p1, p2 = w.pos.copy(), w.pos.copy()
        p1[a, i] += h
        p2[a, i] -= h
        e1 = oracle.compute(w.model, w.params, w.es, p1, w.types, w.box, use_bins=False)["energy"]
        e2 = oracle.compute(w.model, w.params, w.es, p2, w.types, w.box, use_bins=False)["energy"]
        fd = -(e1 - e2) / (2 * h)
        assert abs(fd - out["forces"][a, i]) < 2e-7 * max(1.0, abs(fd)), (fd, out["forces"][a, i])
    for (a, b) in ((0, 0), (1, 1), (0, 2), (2, 1)):
        eps = np.zeros((3, 3))
        eps[a, b] = h
        def energy(sign):
            Fm = np.eye(3) + sign * eps
            return oracle.compute(w.model, w.params, w.es, Fm @ w.pos, w.types,
                                  (w.box.reshape(3, 3) @ Fm.T).ravel(), use_bins=False)["energy"]
        fd = -(energy(1) - energy(-1)) / (2 * h)
        assert abs(fd - out["virial"][a, b]) < 1e-6 * np.abs(out["virial"]).max(), (fd, out["virial"][a, b])
    assert np.abs(out["forces"].sum(axis=1)).max() < 1e-10
    assert np.allclose(out["virial"], out["virial"].T, atol=1e-9 * np.abs(out["virial"]).max())


def test_triclinic_pppm_converges_to_ewald(oracle):
    """Eq. 34-39 with the mesh in fractional coordinates and k from the reciprocal basis vectors (:104): on a triclinic cell the
    PPPM energy, potential, forces, virial and per-atom virial converge to the Ewald sum as the mesh is refined."""
    L = 16.0
    pos, q = _random_charges(120, L, 9)
    h = np.array([[L, 0.0, 0.0], [0.2 * L, L, 0.0], [0.1 * L, -0.15 * L, 0.9 * L]])
    frac = pos / L
    pos = h.T @ frac
    box = h.ravel()
    ew = oracle.electrostatics(pos, q, box, 6.0, 2, I.EsDesc(method=1, alpha=0.3, ewald_nmax2=225), want_atom_virial=True)
    errs = []
    for g in (16, 32, 64):
        pm = oracle.electrostatics(pos, q, box, 6.0, 2, I.EsDesc(method=2, alpha=0.3, grid=(g, g, g)), want_atom_virial=(g == 64))
        errs.append((rel_rms(pm["F"], ew["F"]), abs(pm["U"][1] - ew["U"][1]) / abs(ew["U"][1]),
                     rel_rms(pm["phi"], ew["phi"]), np.abs(pm["W"] - ew["W"]).max() / np.abs(ew["W"]).max()))
    assert errs[0][0] < 2e-3 and errs[1][0] < 2e-5 and errs[2][0] < 2e-7, errs
    assert errs[0][0] > 10 * errs[1][0] > 100 * errs[2][0]
    assert errs[2][1] < 1e-7 and errs[2][2] < 1e-6 and errs[2][3] < 1e-6, errs
    assert rel_rms(pm["W_atom"], ew["W_atom"]) < 1e-5
    # anisotropic mesh on the same cell
    pm2 = oracle.electrostatics(pos, q, box, 6.0, 2, I.EsDesc(method=2, alpha=0.3, grid=(64, 32, 32)))
    assert rel_rms(pm2["F"], ew["F"]) < 3e-5


# --------------------------------------------------- NEP4 4-/5-body terms (reading Z2)
def test_higher_body_descriptors_vs_neighbour_sums(oracle):
    """The 4-body term is a sum over neighbour TRIPLES and the 5-body term a sum over QUADRUPLES of products of the radial
    functions with rotational invariants of the directions (numpy's Chebyshev series, brute-force loops over the neighbours):
        q4_n = sum_jkl g_j g_k g_l [c_jk c_kl c_lj - (c_jk^2 + c_kl^2 + c_lj^2)/3 + 2/9],   q5_n = sum_jklm g_j g_k g_l g_m c_jk c_lm;
    and q4 is the Wigner-3j contraction of the l = 2 moments (complex spherical harmonics from scipy) up to ONE constant."""
    from numpy.polynomial import chebyshev as Ch
    try:
        from scipy.special import sph_harm_y
        Y = lambda l, m, theta, phi: sph_harm_y(l, m, theta, phi)
    except ImportError:
        from scipy.special import sph_harm
        Y = lambda l, m, theta, phi: sph_harm(m, l, phi, theta)
    w = I.with_higher_body_terms(I.config0(), "config0_45body")
    m = w.model
    assert m.n_desc == 35
    p = w.params.astype(np.float64)
    off = I.param_offsets(m)
    nR, nA, Kb = m.n_max_r + 1, m.n_max_a + 1, m.basis_r + 1
    cA = p[off["c_a"]:off["scaler"]].reshape(2, 2, nA, Kb)
    D = oracle.descriptors(m, p, w.pos, w.types, w.box)
    # the first 25 descriptors are those of the plain model with the same coefficients
    w0 = I.config0()
    D0 = oracle.descriptors(w0.model, np.concatenate([p[:off["scaler"]], np.ones(25), np.zeros(w0.model.n_params() - off["scaler"] - 25)]),
                            w.pos, w.types, w.box)
    assert np.allclose(D[:, :25], D0, rtol=1e-13, atol=1e-13)
    counts, jj, dd = oracle.neighbors(w.pos, w.box, m.rc_r, cap=48)

    def g(c, r, rc):
        x = 2 * (r / rc - 1) ** 2 - 1
        fc = 0.5 * (1 + np.cos(np.pi * r / rc))
        return 0.5 * (Ch.chebval(x, c) + c.sum()) * fc

    # Wigner 3j symbols (2 2 2; m1 m2 m3) by the Racah formula
    from math import factorial as f

    def w3j(j1, j2, j3, m1, m2, m3):
        if m1 + m2 + m3 != 0:
            return 0.0
        tri = f(j1 + j2 - j3) * f(j1 - j2 + j3) * f(-j1 + j2 + j3) / f(j1 + j2 + j3 + 1)
        pre = np.sqrt(tri * f(j1 + m1) * f(j1 - m1) * f(j2 + m2) * f(j2 - m2) * f(j3 + m3) * f(j3 - m3))
        tot = 0.0
        for k in range(0, 20):
            den = [k, j1 + j2 - j3 - k, j1 - m1 - k, j2 + m2 - k, j3 - j2 + m1 + k, j3 - j1 - m2 + k]
            if min(den) < 0:
                continue
            tot += (-1) ** k / np.prod([float(f(x)) for x in den])
        return (-1) ** (j1 - j2 - m3) * pre * tot

    ratios = []
    for i in (0, 13, 40):
        ti = w.types[i]
        ang = [(jj[i, s], dd[i, s]) for s in range(counts[i]) if dd[i, s][3] < m.rc_a]
        u = np.array([d[:3] / d[3] for _, d in ang])
        c = u @ u.T
        for n in range(nA):
            gv = np.array([g(cA[ti, w.types[j], n], d[3], m.rc_a) for j, d in ang])
            q4 = np.einsum("j,k,l,jk,kl,lj->", gv, gv, gv, c, c, c) - np.einsum("j,k,l,jk->", gv, gv, gv, c ** 2) + 2.0 / 9.0 * gv.sum() ** 3
            q5 = np.einsum("j,k,jk->", gv, gv, c) ** 2
            assert abs(D[i, 25 + n] - q4) < 1e-10 * max(1.0, abs(q4)), (i, n, D[i, 25 + n], q4)
            assert abs(D[i, 30 + n] - q5) < 1e-10 * max(1.0, abs(q5)), (i, n, D[i, 30 + n], q5)
            A2 = {mm: sum(gj * Y(2, mm, np.arccos(uj[2]), np.arctan2(uj[1], uj[0])) for gj, uj in zip(gv, u)) for mm in range(-2, 3)}
            inv3j = sum(w3j(2, 2, 2, a, b, -a - b) * A2[a] * A2[b] * A2[-a - b] for a in range(-2, 3) for b in range(-2, 3) if abs(a + b) <= 2)
            assert abs(inv3j.imag) < 1e-10 * max(1.0, abs(inv3j.real))
            if abs(q4) > 1e-6:
                ratios.append(inv3j.real / q4)
    assert len(ratios) >= 8 and np.ptp(ratios) < 1e-9 * abs(np.mean(ratios)), ratios     # one constant for all environments


def test_higher_body_terms_invariance_and_derivatives(oracle):
    """With the 4-/5-body terms on: rotation and translation invariance of energy and charges, F = -dE/dr and
    W = -dE/d(strain) by central differences, BEC sum rule, and the new descriptors do move the result."""
    w = I.with_higher_body_terms(_small_workload(2, 0.3), "config0_45body")
    out = oracle.compute_workload(w, use_bins=False, want_bec=True, want_atom_virial=True)
    h = 1e-5
    for (a, i) in ((0, 2), (1, 30), (2, 61)):
        p1, p2 = w.pos.copy(), w.pos.copy()
        p1[a, i] += h
        p2[a, i] -= h
        e1 = oracle.compute(w.model, w.params, w.es, p1, w.types, w.box, use_bins=False)["energy"]
        e2 = oracle.compute(w.model, w.params, w.es, p2, w.types, w.box, use_bins=False)["energy"]
        fd = -(e1 - e2) / (2 * h)
        assert abs(fd - out["forces"][a, i]) < 2e-7 * max(1.0, abs(fd)), (fd, out["forces"][a, i])
    for (a, b) in ((0, 0), (1, 2)):
        eps = np.zeros((3, 3))
        eps[a, b] = h
        def energy(sign):
            Fm = np.eye(3) + sign * eps
            return oracle.compute(w.model, w.params, w.es, Fm @ w.pos, w.types,
                                  (w.box.reshape(3, 3) @ Fm.T).ravel(), use_bins=False)["energy"]
        fd = -(energy(1) - energy(-1)) / (2 * h)
        assert abs(fd - out["virial"][a, b]) < 1e-6 * np.abs(out["virial"]).max(), (fd, out["virial"][a, b])
    assert np.abs(out["forces"].sum(axis=1)).max() < 1e-10
    assert np.allclose(out["virial_atom"].sum(axis=1).reshape(3, 3), out["virial"], atol=1e-9 * np.abs(out["virial"]).max())
    # a rotation that maps the cubic box onto itself (x -> y -> z -> x): energy and charges unchanged, forces rotate
    rot = np.array([[0.0, 0.0, 1.0], [1.0, 0.0, 0.0], [0.0, 1.0, 0.0]])
    r = oracle.compute(w.model, w.params, w.es, rot @ w.pos, w.types, w.box, use_bins=False)
    assert abs(r["energy"] - out["energy"]) < 1e-10 and np.abs(r["charges"] - out["charges"]).max() < 1e-12
    assert np.abs(r["forces"] - rot @ out["forces"]).max() < 1e-10
    # the extra descriptors carry weight: zeroing their scaler changes the energy
    off = I.param_offsets(w.model)
    p0 = w.params.copy()
    p0[off["scaler"] + 25:off["scaler"] + 35] = 0.0
    assert abs(oracle.compute(w.model, p0, w.es, w.pos, w.types, w.box, use_bins=False)["energy"] - out["energy"]) > 1e-4
