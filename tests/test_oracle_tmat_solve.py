"""Pins P7, P8, P9, P11, P13: T symmetry, T vs F cross-check,
two-/three-site closed forms, dense Cholesky vs PCG, energy identities."""
import numpy as np
import pytest

import oracle
from synth_inputs import System, make_config, tiny_cluster, water_box

A_THOLE = 0.39


def _sites(pos, alpha, box=0.0, rc=50.0, beta=0.0):
    pos = np.asarray(pos, float).reshape(-1, 3)
    n = pos.shape[0]
    return System(name="sites", box=box, pos=pos, charge=np.zeros(n), dipole=np.zeros((n, 3)),
                  quad=np.zeros((n, 6)), polarizability=np.asarray(alpha, float),
                  group_id=np.arange(n, dtype=np.int32), cutoff=rc, skin=0.0,
                  ewald_beta=beta, thole_a=A_THOLE)


def test_p7_T_is_symmetric_bilinear():
    s = make_config(0)
    rng = np.random.default_rng(1)
    mu, nu = rng.standard_normal((2, s.n_atoms, 3))
    a = float(np.sum(nu * oracle.tmatvec(s, mu)))
    b = float(np.sum(mu * oracle.tmatvec(s, nu)))
    assert abs(a - b) <= 1e-13 * max(abs(a), abs(b))


def test_p7_T_equals_field_of_pure_dipoles():
    """T mu == F applied with q = 0, Theta = 0, d = mu and no masks (two separately
    written routines: tmu_row and field_row)."""
    s = make_config(0)
    rng = np.random.default_rng(2)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    as_field = s.with_(charge=np.zeros(s.n_atoms), quad=np.zeros((s.n_atoms, 6)), dipole=mu,
                       group_id=np.arange(s.n_atoms, dtype=np.int32))
    np.testing.assert_allclose(oracle.tmatvec(s, mu), oracle.perm_field(as_field),
                               rtol=1e-12, atol=1e-14)


def test_p7_dense_T_symmetric_and_matches_matvec():
    s = tiny_cluster(40, 3, box=14.0, spread=14.0, cutoff=6.5, ewald_beta=0.55)
    T = oracle.dense_T(s)
    assert np.abs(T - T.T).max() <= 2e-16 * np.abs(T).max() + 1e-18
    rng = np.random.default_rng(4)
    mu = rng.standard_normal((s.n_atoms, 3))
    np.testing.assert_allclose((T @ mu.reshape(-1)).reshape(-1, 3), oracle.tmatvec(s, mu),
                               rtol=1e-12, atol=1e-13)
    rows = np.array([3, 39, 0])
    np.testing.assert_array_equal(oracle.tmatvec_rows(s, mu, rows), oracle.tmatvec(s, mu)[rows])


@pytest.mark.parametrize("direction", ["par", "perp"])
def test_p8_two_site_closed_form(golden, direction):
    g = golden["P8_two_site"]
    R, E0 = g["R"], g["E"]
    s = _sites([[0, 0, 0], [0, 0, R]], g["alpha"])
    axis = np.array([0, 0, 1.0]) if direction == "par" else np.array([1.0, 0, 0])
    E = np.tile(E0 * axis, (2, 1))
    # coupling constants from the oracle's T
    T = oracle.dense_T(s)
    k = 2 if direction == "par" else 0
    assert T[k, 3 + k] == pytest.approx(g["t_" + direction], rel=1e-13)
    mu_ref = np.array(g["mu_" + direction])
    for mu in (oracle.dense_solve(s, E), oracle.pcg_solve(s, E, tol=1e-14)[0]):
        np.testing.assert_allclose(mu @ axis, mu_ref, rtol=1e-12)
        off = mu - np.outer(mu @ axis, axis)
        assert np.abs(off).max() < 1e-16
        assert oracle.polar_energy(mu, E) == pytest.approx(g["Epol_" + direction], rel=1e-12)
    # textbook formula mu1 = a1 (E1 + t a2 E2) / (1 - a1 a2 t^2), written out here
    a1, a2 = g["alpha"]
    t = g["t_" + direction]
    np.testing.assert_allclose(mu_ref, [a1 * E0 * (1 + t * a2) / (1 - a1 * a2 * t * t),
                                        a2 * E0 * (1 + t * a1) / (1 - a1 * a2 * t * t)],
                               rtol=1e-13)


@pytest.mark.parametrize("shape", ["collinear", "equilateral"])
def test_p9_three_site(shape):
    if shape == "collinear":
        pos = [[0, 0, 0], [0, 0, 1.9], [0, 0, 4.1]]
    else:
        pos = [[0, 0, 0], [2.2, 0, 0], [1.1, 2.2 * np.sqrt(3) / 2, 0]]
    s = _sites(pos, [0.837, 0.496, 1.3])
    rng = np.random.default_rng(7)
    E = rng.standard_normal((3, 3)) * 0.1
    mu_d = oracle.dense_solve(s, E)
    mu_p, it, rms = oracle.pcg_solve(s, E, tol=1e-13)
    np.testing.assert_allclose(mu_p, mu_d, rtol=1e-10, atol=1e-14)
    # residual recomputed from scratch
    res = E - (mu_d / s.polarizability[:, None] - oracle.tmatvec(s, mu_d))
    assert np.abs(res).max() < 1e-14
    if shape == "collinear":
        # a field along the axis induces dipoles along the axis only
        Ez = np.zeros((3, 3)); Ez[:, 2] = 0.1
        mz = oracle.dense_solve(s, Ez)
        assert np.abs(mz[:, :2]).max() < 1e-16 and np.all(mz[:, 2] > 0)


def test_p9_water_box_pcg_vs_cholesky():
    s = make_config(0)
    E = oracle.perm_field(s)
    A = oracle.dense_A(s)
    w = np.linalg.eigvalsh(A)
    assert w[0] > 0.5, "A must be SPD"
    mu_d = oracle.dense_solve(s, E)
    mu_p, it, rms = oracle.pcg_solve(s, E, tol=1e-12)
    assert np.linalg.norm(mu_p - mu_d) <= 1e-10 * np.linalg.norm(mu_d)
    # P13 sanity on iteration counts (not parity)
    for tol, lo, hi in ((1e-5, 4, 9), (1e-6, 6, 11), (1e-8, 9, 15)):
        _, it, rms = oracle.pcg_solve(s, E, tol=tol)
        assert lo <= it <= hi and rms < tol


def test_p9_solute_mixture_is_spd():
    s = water_box(512, 24.85, 77, solute_frac=0.15)
    A = oracle.dense_A(s)
    assert np.linalg.eigvalsh(A)[0] > 0.1
    E = oracle.perm_field(s)
    mu_d = oracle.dense_solve(s, E)
    mu_p, it, _ = oracle.pcg_solve(s, E, tol=1e-12)
    assert np.linalg.norm(mu_p - mu_d) <= 1e-10 * np.linalg.norm(mu_d)


def test_p11_energy_is_minimum_of_quadratic_and_gradient_wrt_field():
    s = tiny_cluster(33, 21, box=13.0, spread=13.0, cutoff=6.0, ewald_beta=0.6)
    E = oracle.perm_field(s)
    mu = oracle.dense_solve(s, E)
    A = oracle.dense_A(s)
    f = oracle.COULOMB
    W = f * (0.5 * mu.reshape(-1) @ A @ mu.reshape(-1) - np.sum(mu * E))
    assert oracle.polar_energy(mu, E) == pytest.approx(W, rel=1e-12)
    # any other mu has higher W
    rng = np.random.default_rng(0)
    mu2 = mu + 1e-3 * rng.standard_normal(mu.shape)
    W2 = f * (0.5 * mu2.reshape(-1) @ A @ mu2.reshape(-1) - np.sum(mu2 * E))
    assert W2 > W
    # dE_pol/dE_i = -f mu_i (central differences of the right-hand side)
    h = 1e-5
    for (i, c) in ((0, 0), (17, 2), (32, 1)):
        Ep, Em = E.copy(), E.copy()
        Ep[i, c] += h
        Em[i, c] -= h
        ep = oracle.polar_energy(oracle.dense_solve(s, Ep), Ep)
        em = oracle.polar_energy(oracle.dense_solve(s, Em), Em)
        assert (ep - em) / (2 * h) == pytest.approx(-f * mu[i, c], rel=1e-7)


def test_pcg_guess_and_iteration_cap():
    s = make_config(0)
    E = oracle.perm_field(s)
    mu, it, rms = oracle.pcg_solve(s, E, tol=1e-9)
    mu2, it2, rms2 = oracle.pcg_solve(s, E, tol=1e-9, guess=mu)
    assert it2 == 0 and rms2 < 1e-9
    _, it3, rms3 = oracle.pcg_solve(s, E, tol=1e-30, max_iter=3)
    assert it3 == 3 and rms3 > 1e-30


def test_pair_count_matches_density():
    s = make_config(0)
    n_pair = oracle.count_pairs(s)
    # (4/3) pi rc^3 rho / 2 per atom, rho = N / L^3  (~71-72 at 7 A)
    expect = 0.5 * 4 / 3 * np.pi * s.cutoff**3 * s.n_atoms / s.box**3
    assert abs(n_pair / s.n_atoms - expect) < 0.03 * expect
    rows = np.arange(0, s.n_atoms, 5)
    tot = oracle.count_pairs_rows(s, np.arange(s.n_atoms))
    assert tot == 2 * n_pair
    assert oracle.count_pairs_rows(s, rows) > 0


def _brute_force_pairs(pos, box, cutoff):
    """The definition, written out here in numpy (not through oracle/): unordered pairs i < j with
    minimum-image R^2 <= r_c^2, and the same count per row."""
    n = pos.shape[0]
    d = pos[:, None, :] - pos[None, :, :]
    if box > 0:
        d = d - box * np.rint(d / box)
    r2 = np.einsum("ijk,ijk->ij", d, d)
    inside = r2 <= cutoff * cutoff
    np.fill_diagonal(inside, False)
    return int(np.triu(inside, 1).sum()), inside.sum(axis=1)


@pytest.mark.parametrize("periodic", [True, False])
def test_pair_count_is_exact_against_brute_force(periodic):
    """SURVEY 8(c) Q7 (R^2 <= r_c^2, inclusive) and Q17 (single minimum image): count_pairs and
    count_pairs_rows against a numpy brute force, with one pair placed exactly on the cutoff and, in
    the periodic case, one pair that is only inside r_c through the boundary.  A `<` written for
    `<=` or a dropped minimum image fails here."""
    from synth_inputs import tiny_cluster
    if periodic:
        s = tiny_cluster(65, 11, box=14.0, spread=14.0, cutoff=5.0, skin=1.0, ewald_beta=0.6)
    else:
        s = tiny_cluster(97, 12, box=0.0, spread=12.0, cutoff=5.0, skin=1.0)
    pos = s.pos.copy()
    # atoms 0 and 1 exactly r_c apart along x (1.0 and 6.0 are exact in FP64: R^2 == r_c^2 == 25)
    pos[0] = (1.0, 3.25, 7.5)
    pos[1] = (6.0, 3.25, 7.5)
    if periodic:
        # atoms 2 and 3: 13.0 apart in the box, 1.0 apart through the boundary
        pos[2] = (0.25, 9.0, 2.0)
        pos[3] = (13.25, 9.0, 2.0)
    s = s.with_(pos=pos)
    n_ref, per_row = _brute_force_pairs(pos, s.box, s.cutoff)
    d01 = pos[0] - pos[1]
    assert float(d01 @ d01) == s.cutoff ** 2                   # the edge pair really sits on the edge
    assert oracle.count_pairs(s) == n_ref
    rows = np.array([0, 1, 2, 3, 17, 40, s.n_atoms - 1], dtype=np.int64)
    assert oracle.count_pairs_rows(s, rows) == int(per_row[rows].sum())
    assert oracle.count_pairs_rows(s, np.arange(s.n_atoms)) == 2 * n_ref == int(per_row.sum())
    # the edge pair and (periodic) the boundary pair are among the counted ones
    assert oracle.count_pairs_rows(s, np.array([0])) == int(per_row[0]) >= 1
    if periodic:
        no_image = _brute_force_pairs(pos, 0.0, s.cutoff)[0]
        assert no_image < n_ref                                # the minimum image matters in this system
