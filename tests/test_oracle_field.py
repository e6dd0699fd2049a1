"""Pins P3, P4, P5, P6, P10 for the permanent field (F1-F3).

The scalar potentials used here are written out in this file from (F4) with
scipy special functions; they share nothing with oracle/."""
import numpy as np
import pytest
from scipy.special import erfc, gamma, gammaincc

import oracle
from synth_inputs import System, make_config, tiny_cluster

A_THOLE = 0.39


def _system(pos, q=None, dip=None, quad=None, alpha=None, grp=None, box=0.0,
            rc=50.0, beta=0.0):
    pos = np.asarray(pos, dtype=np.float64).reshape(-1, 3)
    n = pos.shape[0]
    z = np.zeros
    return System(name="t", box=box, pos=pos,
                  charge=z(n) if q is None else np.asarray(q, float),
                  dipole=z((n, 3)) if dip is None else np.asarray(dip, float).reshape(n, 3),
                  quad=z((n, 6)) if quad is None else np.asarray(quad, float).reshape(n, 6),
                  polarizability=np.ones(n) if alpha is None else np.asarray(alpha, float),
                  group_id=np.arange(n, dtype=np.int32) if grp is None else np.asarray(grp, np.int32),
                  cutoff=rc, skin=0.0, ewald_beta=beta, thole_a=A_THOLE)


def _pair_kernel(R, beta, ai, aj, s):
    """f(R) with -f'/R = G1 (F4): erfc(bR)/R - 1/R + s [lambda3/R + c^(1/3) Gamma(2/3,cR^3)]."""
    c = A_THOLE / np.sqrt(ai * aj)
    x = c * R**3
    g = (1 - np.exp(-x)) / R + c ** (1 / 3) * gammaincc(2 / 3, x) * gamma(2 / 3)
    ew = erfc(beta * R) / R if beta > 0 else 1.0 / R
    return ew - 1.0 / R + s * g


def test_p4_single_charge_closed_form(golden):
    g = golden["P4_charge_field"]
    s = _system([[0, 0, 0], [2.0, 0, 0]], q=[0.0, -1.0], alpha=g["alpha"], beta=g["beta"])
    E = oracle.perm_field(s)
    assert E[0, 0] == pytest.approx(g["Ex_at_origin"], rel=1e-12)
    assert abs(E[0, 1]) < 1e-16 and abs(E[0, 2]) < 1e-16
    assert np.all(E[1] == 0.0)  # the source carries the only multipole


def test_p5_isolated_molecule_has_zero_field():
    """Open boundary, beta = 0: every intramolecular pair is masked, G_k = 0."""
    w = make_config(0)
    mol = _system(w.pos[:3], q=w.charge[:3], dip=w.dipole[:3], quad=w.quad[:3],
                  alpha=w.polarizability[:3], grp=[0, 0, 0])
    E = oracle.perm_field(mol)
    assert np.all(np.abs(E) < 1e-13)
    # same three atoms as three groups: field is non-zero
    E2 = oracle.perm_field(mol.with_(group_id=np.array([0, 1, 2], np.int32)))
    assert np.abs(E2).max() > 1e-2


@pytest.mark.parametrize("beta,s", [(0.0, 1), (0.5446, 1), (0.5446, 0)])
def test_p6_charge_field_is_minus_gradient_of_potential(beta, s):
    rng = np.random.default_rng(5)
    rj = np.array([0.3, -0.2, 0.1])
    ri = rj + np.array([1.1, 0.7, -0.9])
    ai, aj, qj = 0.837, 0.496, 0.73
    grp = [0, 0] if s == 0 else [0, 1]
    sysm = _system([ri, rj], q=[0.0, qj], alpha=[ai, aj], grp=grp, beta=beta)
    E = oracle.perm_field(sysm)[0]

    def phi(p):
        return qj * _pair_kernel(np.linalg.norm(p - rj), beta, ai, aj, s)

    h = 1e-4
    grad = np.array([(phi(ri + h * e) - phi(ri - h * e)) / (2 * h) for e in np.eye(3)])
    # Richardson with 2h
    grad2 = np.array([(phi(ri + 2 * h * e) - phi(ri - 2 * h * e)) / (4 * h) for e in np.eye(3)])
    grad = (4 * grad - grad2) / 3
    np.testing.assert_allclose(E, -grad, rtol=2e-9, atol=1e-12)
    del rng


def _field_at(probe, src_pos, q=None, dip=None, quad=None, beta=0.5446, alpha=(0.837, 0.496),
              masked=False, box=0.0, rc=50.0):
    """Field at one probe point from ONE multipolar source (probe carries nothing)."""
    grp = [0, 0] if masked else [0, 1]
    sysm = _system([probe, src_pos], q=[0.0, 0.0 if q is None else q],
                   dip=None if dip is None else [np.zeros(3), dip],
                   quad=None if quad is None else [np.zeros(6), quad],
                   alpha=alpha, grp=grp, beta=beta, box=box, rc=rc)
    return oracle.perm_field(sysm)[0]


@pytest.mark.parametrize("masked", [False, True])
@pytest.mark.parametrize("beta", [0.0, 0.5446])
def test_p6_dipole_and_quadrupole_fields_are_gradients(beta, masked):
    """phi_dip = (d.R) G1(R),  phi_quad = (1/3)(R.Theta R) G2(R)  (F4), E = -grad phi.
    G1, G2 come from oracle.pair_G, which test_oracle_radial pins independently."""
    rj = np.array([0.2, 0.1, -0.3])
    ri = rj + np.array([-1.3, 0.8, 1.0])
    ai, aj = 0.837, 0.496
    d = np.array([0.21, -0.4, 0.33])
    th = np.array([0.3, -0.1, 0.25, -0.45, 0.12, 0.15])  # xx xy xz yy yz zz, traceless
    TH = np.array([[th[0], th[1], th[2]], [th[1], th[3], th[4]], [th[2], th[4], th[5]]])
    s = 0.0 if masked else 1.0

    def G(p):
        R = np.linalg.norm(p - rj)
        return oracle.pair_G(beta, A_THOLE, ai, aj, s, R)

    def phi_d(p):
        return float(d @ (p - rj)) * G(p)[0]

    def phi_q(p):
        R = p - rj
        return float(R @ TH @ R) * G(p)[1] / 3.0

    def minus_grad(phi):
        h = 1e-4
        g1 = np.array([(phi(ri + h * e) - phi(ri - h * e)) / (2 * h) for e in np.eye(3)])
        g2 = np.array([(phi(ri + 2 * h * e) - phi(ri - 2 * h * e)) / (4 * h) for e in np.eye(3)])
        return -(4 * g1 - g2) / 3

    Ed = _field_at(ri, rj, dip=d, beta=beta, masked=masked)
    Eq = _field_at(ri, rj, quad=th, beta=beta, masked=masked)
    np.testing.assert_allclose(Ed, minus_grad(phi_d), rtol=5e-9, atol=1e-12)
    np.testing.assert_allclose(Eq, minus_grad(phi_q), rtol=5e-9, atol=1e-12)


@pytest.mark.parametrize("beta", [0.0, 0.5446])
def test_p3_dipole_is_limit_of_two_charges(beta):
    """Point-charge-cluster limit: +-q at +-delta/2 along d, all carrying the source's
    alpha; the CHARGE path (closed form q G1 R, pin P4) must reproduce the dipole
    path as delta -> 0 (error O(delta^2), Richardson-extrapolated)."""
    probe = np.array([1.4, -0.9, 1.2])
    src = np.array([0.1, 0.2, -0.1])
    d = np.array([0.3, -0.2, 0.45])
    dn = np.linalg.norm(d)
    u = d / dn

    def cluster(delta):
        q = dn / delta
        sysm = _system([probe, src + 0.5 * delta * u, src - 0.5 * delta * u],
                       q=[0.0, q, -q], alpha=[0.837, 0.496, 0.496], grp=[0, 1, 1], beta=beta)
        return oracle.perm_field(sysm)[0]

    e1, e2 = cluster(2e-3), cluster(1e-3)
    extrap = (4 * e2 - e1) / 3
    want = _field_at(probe, src, dip=d, beta=beta)
    np.testing.assert_allclose(extrap, want, rtol=2e-8, atol=1e-12)


@pytest.mark.parametrize("beta", [0.0, 0.5446])
def test_p3_quadrupole_is_limit_of_charge_cluster(beta):
    """Theta = 1/2 sum q (3 r r^T - r^2 I)  (Q2, F4).  Cluster: for each Cartesian pair
    a general traceless Theta is built from axial (+q,-2q,+q) linear quadrupoles along
    three directions; here: charges on the 6 face points +-delta e_k with weights w_k and
    a centre charge -2 sum w_k, plus 4 diagonal points for each off-diagonal element."""
    probe = np.array([1.5, 1.1, -1.3])
    src = np.array([-0.1, 0.15, 0.2])

    def cluster_field(delta):
        pts, qs = [], []
        # diagonal part: charges w_k at +-delta e_k  -> Theta_kk contribution
        # 1/2 * 2 w_k (3 delta^2 - delta^2) = 2 w_k delta^2 on kk, -w_k delta^2 on the others
        w = np.array([0.7, -0.2, -0.5]) / delta**2
        for k in range(3):
            for sgn in (+1, -1):
                pts.append(src + sgn * delta * np.eye(3)[k])
                qs.append(w[k])
        # off-diagonal xy: charges +-v at (+-delta, +-delta, 0):  Theta_xy = 1/2 * 3 * 4 v delta^2
        v = 0.31 / delta**2
        for sx in (+1, -1):
            for sy in (+1, -1):
                pts.append(src + delta * np.array([sx, sy, 0.0]))
                qs.append(v * sx * sy)
        pts.append(src)
        qs.append(-2 * w.sum())  # neutral; off-diagonal set is neutral already
        n = len(pts) + 1
        sysm = _system([probe] + pts, q=[0.0] + qs, alpha=[0.837] + [0.496] * (n - 1),
                       grp=[0] + [1] * (n - 1), beta=beta)
        return oracle.perm_field(sysm)[0]

    wq = np.array([0.7, -0.2, -0.5])
    diag = 2 * wq - (wq.sum() - wq)          # Theta_kk = 2 w_k - sum_{m != k} w_m (delta^2 = 1 units)
    th = np.array([diag[0], 6 * 0.31, 0.0, diag[1], 0.0, diag[2]])
    # the xy charges also add to the diagonal: 1/2 sum q (3 x^2 - r^2) = 0 since sum q = 0 and x^2 equal
    assert abs(th[0] + th[3] + th[5]) < 1e-12
    e1, e2 = cluster_field(4e-3), cluster_field(2e-3)
    extrap = (4 * e2 - e1) / 3
    want = _field_at(probe, src, quad=th, beta=beta)
    np.testing.assert_allclose(extrap, want, rtol=5e-7, atol=1e-11)


def test_self_term_and_cutoff():
    """(F3) self term 4 b^3/(3 sqrt(pi)) d_i ; (Q7) pairs beyond rc contribute nothing."""
    beta = 0.5446
    d = np.array([0.1, -0.3, 0.2])
    lone = _system([[0, 0, 0], [30.0, 0, 0]], dip=[d, np.zeros(3)], beta=beta, rc=7.0)
    E = oracle.perm_field(lone)
    np.testing.assert_allclose(E[0], 4 * beta**3 / (3 * np.sqrt(np.pi)) * d, rtol=1e-15)
    assert np.all(E[1] == 0.0)
    # R^2 <= rc^2 is inclusive
    edge = _system([[0, 0, 0], [7.0, 0, 0]], q=[0, 1.0], beta=beta, rc=7.0)
    assert oracle.perm_field(edge)[0, 0] != 0.0
    out = _system([[0, 0, 0], [np.nextafter(7.0, 8.0), 0, 0]], q=[0, 1.0], beta=beta, rc=7.0)
    assert oracle.perm_field(out)[0, 0] == 0.0


def test_p10_invariances():
    s = make_config(0)
    E0 = oracle.perm_field(s)
    # translate everything
    E1 = oracle.perm_field(s.with_(pos=s.pos + np.array([3.7, -11.2, 40.05])))
    np.testing.assert_allclose(E1, E0, rtol=0, atol=2e-12)
    # shift individual atoms by +-L (breaks molecules across images)
    rng = np.random.default_rng(3)
    shift = rng.integers(-2, 3, size=s.pos.shape) * s.box
    E2 = oracle.perm_field(s.with_(pos=s.pos + shift))
    np.testing.assert_allclose(E2, E0, rtol=0, atol=2e-12)
    # permute atom order: outputs permute
    p = rng.permutation(s.n_atoms)
    sp = s.with_(pos=s.pos[p], charge=s.charge[p], dipole=s.dipole[p], quad=s.quad[p],
                 polarizability=s.polarizability[p], group_id=s.group_id[p])
    E3 = oracle.perm_field(sp)
    np.testing.assert_allclose(E3, E0[p], rtol=0, atol=2e-12)


def test_periodic_image_is_used():
    """A source just across the periodic boundary acts through its nearest image."""
    L = 20.0
    a = _system([[0.5, 5, 5], [19.5, 5, 5]], q=[0, 1.0], box=L, rc=7.0, beta=0.5446)
    b = _system([[0.5, 5, 5], [-0.5, 5, 5]], q=[0, 1.0], box=0.0, rc=7.0, beta=0.5446)
    np.testing.assert_allclose(oracle.perm_field(a)[0], oracle.perm_field(b)[0], rtol=1e-13)


def test_rows_variant_matches_full():
    s = tiny_cluster(65, 11, box=12.0, spread=12.0, cutoff=5.0, ewald_beta=0.6)
    E = oracle.perm_field(s)
    rows = np.array([0, 7, 33, 64])
    np.testing.assert_array_equal(oracle.perm_field_rows(s, rows), E[rows])
