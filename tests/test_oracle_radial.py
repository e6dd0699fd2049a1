"""Pins P1, P2, P5: the oracle's radial functions against
(a) closed-form values recorded in tests/golden/survey_pins.json and
(b) their definitions as derivatives, evaluated with mpmath at 40 digits --
neither route uses any oracle code."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle

mp.mp.dps = 40


def test_p1_bn_golden(golden):
    g = golden["P1_ewald_bn"]
    for case in g["cases"]:
        got = oracle.ewald_bn(g["beta"], case["R"])
        np.testing.assert_allclose(got, case["bn"], rtol=2e-13, atol=0)


@pytest.mark.parametrize("R", [0.8, 0.9572, 1.7, 2.3, 4.4, 6.9])
@pytest.mark.parametrize("beta", [0.5446, 0.31768, 0.9])
def test_p1_bn_is_iterated_derivative(beta, R):
    """bn_k = (-(1/R) d/dR)^k [erfc(beta R)/R]  (definition)."""
    b = mp.mpf(beta)

    def f0(r):
        return mp.erfc(b * r) / r

    def step(f):
        return lambda r: -mp.diff(f, r) / r

    fs = [f0]
    for _ in range(3):
        fs.append(step(fs[-1]))
    want = [float(f(mp.mpf(R))) for f in fs]
    got = oracle.ewald_bn(beta, R)
    np.testing.assert_allclose(got, want, rtol=5e-12)


@pytest.mark.parametrize("R", [0.5, 1.3, 7.0])
def test_p1_beta_zero_is_bare_coulomb(R):
    got = oracle.ewald_bn(0.0, R)
    want = [1 / R, 1 / R**3, 3 / R**5, 15 / R**7]
    np.testing.assert_allclose(got, want, rtol=1e-15)
    # and the beta -> 0 limit of the screened form approaches it
    near = oracle.ewald_bn(1e-4, R)
    np.testing.assert_allclose(near[1:], want[1:], rtol=1e-9)


def test_p2_lambda_golden(golden):
    g = golden["P2_thole_lambda"]
    for case in g["cases"]:
        got = oracle.thole_lambda(g["a"], case["alpha"][0], case["alpha"][1], case["R"])
        np.testing.assert_allclose(got, case["lambda"], rtol=2e-13)


@pytest.mark.parametrize("R", [0.6, 0.9572, 1.5139, 2.4, 3.9])
def test_p2_lambda_derivative_identities(R):
    """lambda_5 = lambda_3 - R lambda_3'/3 ; lambda_7 = lambda_5 - R lambda_5'/5
    (the three are successive radial derivatives of ONE damped kernel)."""
    a, ai, aj = 0.39, 0.837, 0.496
    c = mp.mpf(a) / mp.sqrt(mp.mpf(ai) * mp.mpf(aj))

    def l3(r):
        return 1 - mp.exp(-c * r**3)

    def l5(r):
        return l3(r) - r * mp.diff(l3, r) / 3

    def l7(r):
        return l5(r) - r * mp.diff(l5, r) / 5

    want = [float(l3(mp.mpf(R))), float(l5(mp.mpf(R))), float(l7(mp.mpf(R)))]
    got = oracle.thole_lambda(a, ai, aj, R)
    np.testing.assert_allclose(got, want, rtol=1e-11, atol=1e-15)


def test_p2_lambda_limits():
    far = oracle.thole_lambda(0.39, 0.837, 0.496, 9.0)
    np.testing.assert_allclose(far, [1, 1, 1], atol=1e-15)
    near = oracle.thole_lambda(0.39, 0.837, 0.496, 1e-3)
    assert np.all(np.abs(near) < 1e-8)
    # symmetric in the two polarizabilities
    np.testing.assert_array_equal(oracle.thole_lambda(0.39, 0.3, 1.7, 1.4),
                                  oracle.thole_lambda(0.39, 1.7, 0.3, 1.4))


def test_p5_masked_G_golden(golden):
    g = golden["P5_masked_G"]
    got = oracle.pair_G(g["beta"], g["a"], g["alpha"][0], g["alpha"][1], 0.0, g["R"])
    np.testing.assert_allclose(got, g["G"], rtol=5e-13)
    # masked branch is exactly bn_k - rr_k: no alpha dependence
    other = oracle.pair_G(g["beta"], g["a"], 1.7, 0.31, 0.0, g["R"])
    np.testing.assert_array_equal(got, other)


def test_p4_G1_golden(golden):
    g = golden["P4_charge_field"]
    got = oracle.pair_G(g["beta"], g["a"], g["alpha"][0], g["alpha"][1], 1.0, g["R"])
    assert math.isclose(got[0], g["G1"], rel_tol=5e-13)


@pytest.mark.parametrize("s", [0.0, 1.0])
@pytest.mark.parametrize("R", [0.9572, 1.6, 3.1, 6.5])
def test_G_is_iterated_derivative_of_one_kernel(s, R):
    """-f'/R = G1, -G1'/R = G2, -G2'/R = G3 with the scalar pair kernel
    f(R) = erfc(bR)/R - 1/R + s g(R),  g = lambda_3/R + c^(1/3) Gamma(2/3, c R^3)
    (g is the potential whose radial derivative gives lambda_3/R^2; (F4))."""
    beta, a, ai, aj = 0.5446, 0.39, 0.837, 0.496
    b = mp.mpf(beta)
    c = mp.mpf(a) / mp.sqrt(mp.mpf(ai) * mp.mpf(aj))

    def f(r):
        x = c * r**3
        g = (1 - mp.exp(-x)) / r + c ** (mp.mpf(1) / 3) * mp.gammainc(mp.mpf(2) / 3, x)
        return mp.erfc(b * r) / r - 1 / r + s * g

    def step(fn):
        return lambda r: -mp.diff(fn, r) / r

    g1 = step(f)
    g2 = step(g1)
    g3 = step(g2)
    want = [float(g1(mp.mpf(R))), float(g2(mp.mpf(R))), float(g3(mp.mpf(R)))]
    got = oracle.pair_G(beta, a, ai, aj, s, R)
    np.testing.assert_allclose(got, want, rtol=2e-9, atol=1e-16)


def test_fixed_point_containers_eqs_2_and_3():
    """Paper eqs (2)-(3): a = int(round(x 2^fB)), x = real(a) / 2^fB, with the paper's
    numbers: 34 fractional bits for vectors leave 30 for the integer part ("absolute limit 2^29"),
    30 fractional bits for the energy, and "27 bits ... capture 8 digits after the decimal point"."""
    import oracle as o
    assert o.FIX_VEC_BITS == 34 and o.FIX_ENERGY_BITS == 30
    assert int(o.to_fixed(1.0, 34)) == 1 << 34 and int(o.to_fixed(-0.5, 30)) == -(1 << 29)
    assert float(o.from_fixed(1 << 34, 34)) == 1.0
    # the container holds |x| < 2^29 with 34 fractional bits (63 value bits)
    assert int(o.to_fixed(2.0 ** 29 - 1.0, 34)) < 2 ** 63
    # resolution: half a unit in the last place of the container
    rng = np.random.default_rng(3)
    x = rng.uniform(-100.0, 100.0, 1000)
    for fb in (27, 30, 34):
        back = o.from_fixed(o.to_fixed(x, fb), fb)
        assert np.max(np.abs(back - x)) <= 2.0 ** -(fb + 1)
        assert np.all(o.to_fixed(back, fb) == o.to_fixed(x, fb))          # idempotent
    assert 2.0 ** -27 < 1e-8 < 2.0 ** -26                                  # 27 bits <-> 8 decimal digits
    # integer sums are order independent (what makes the mode deterministic)
    a = o.to_fixed(rng.standard_normal(4096) * 1e-3, 34)
    assert int(a.sum()) == int(a[::-1].sum()) == int(np.sort(a).sum())


def test_fixed_point_energy_converts_one_term_per_atom():
    """polar_energy_fixed (Q21): the sum of per-atom terms rounded to 2^-30 kcal/mol.  Pins:
    a hand-made case whose terms are exact multiples of 2^-30 (nothing is rounded: equals -1/2 f sum mu.E
    computed in exact rational arithmetic); a term of 0.4 units rounds to 0 PER ATOM (three components of
    0.4 units each would round to 0 + 0 + 0 = 0 as well, but 1.2 units per atom must give 1: this is what
    separates per-atom from per-component conversion); the distance to the FP64 energy is at most half a
    unit per atom; the value does not depend on the order of the atoms."""
    import oracle as o
    from fractions import Fraction
    unit = 2.0 ** -30
    f = Fraction(o.COULOMB)                                  # the double, exactly
    # two atoms with mu.E = 1 exactly (the other components multiply zeros): two equal terms, each the integer
    # nearest to -f/2 x 2^30, found here in rational arithmetic from the bits of the double f
    mu = np.array([[2.0, 0.0, 0.0], [0.0, 4.0, 0.0]])
    E = np.array([[0.5, 9.0, 9.0], [7.0, 0.25, 7.0]])       # dots: 1.0 and 1.0
    exact_units = -f / 2 * 2 ** 30
    nearest = int(exact_units - Fraction(1, 2)) if exact_units < 0 else int(exact_units + Fraction(1, 2))
    assert abs(Fraction(nearest) - exact_units) < Fraction(1, 2)                 # no tie: the nearest integer is unique
    want = Fraction(2 * nearest, 2 ** 30)
    assert Fraction(o.polar_energy_fixed(mu, E)) == want
    # per-atom, not per-component: each component contributes 0.4 units, the atom 1.2 units -> 1 unit
    c = 0.4 * unit / (0.5 * o.COULOMB)                       # |mu_k E_k| worth 0.4 units of energy
    mu1 = np.full((5, 3), 1.0)
    E1 = np.full((5, 3), -c)                                 # energy term +1.2 units per atom
    got = o.polar_energy_fixed(mu1, E1)
    assert got == 5 * unit                                   # per-component rounding would give 0
    # half a unit per atom at most, and order independence
    rng = np.random.default_rng(11)
    mu2 = rng.standard_normal((777, 3)) * 0.05
    E2 = rng.standard_normal((777, 3)) * 0.1
    e_fix = o.polar_energy_fixed(mu2, E2)
    assert abs(e_fix - o.polar_energy(mu2, E2)) <= 777 * 0.5 * unit + 1e-12
    assert e_fix * 2.0 ** 30 == np.rint(e_fix * 2.0 ** 30)
    perm = rng.permutation(777)
    assert o.polar_energy_fixed(mu2[perm], E2[perm]) == e_fix
