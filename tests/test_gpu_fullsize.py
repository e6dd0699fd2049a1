"""GPU parity at BASELINE.json's full sizes (configs 1, 2, 3 and the config-4 sweep), in the launch configuration
bench.py times: sampled rows the oracle computes one by one, the bit-exact block-pair set,
the useful-pair count, and properties that hold at any size."""
import numpy as np
import pytest

import oracle
from synth_inputs import make_config

pytestmark = pytest.mark.gpu


def _rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(b))


def _assert_close(got, ref, tol):
    """BASELINE.json's bar (relative L2 over the compared rows) plus a per-row guard, so that an error
    confined to a few atoms cannot hide in the norm: max_i |got_i - ref_i| <= 50 tol rms_i |ref_i|."""
    got, ref = np.asarray(got, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape
    rel = float(np.linalg.norm(got - ref) / np.linalg.norm(ref))
    assert rel <= tol, f"rel-L2 {rel:.3e} > {tol:.1e}"
    row = np.linalg.norm((got - ref).reshape(ref.shape[0], -1), axis=1)
    rms = float(np.sqrt(np.mean(np.sum(ref.reshape(ref.shape[0], -1) ** 2, axis=1))))
    worst = int(np.argmax(row))
    assert row[worst] <= 50.0 * tol * rms, f"row {worst}: |delta| {row[worst]:.3e} > 50 x {tol:.1e} x rms {rms:.3e}"


@pytest.fixture(scope="module")
def cfg1():
    return make_config(1)


@pytest.fixture(scope="module")
def cfg2():
    return make_config(2)


def _rows(s, perm, n_rand=512, n_blocks=4, seed=0):
    rng = np.random.default_rng(seed)
    rows = set(rng.choice(s.n_atoms, size=n_rand, replace=False).tolist())
    nb = perm.size // 32
    for b in rng.choice(nb, size=n_blocks, replace=False):
        rows.update(int(a) for a in perm[32 * b:32 * b + 32] if a >= 0)
    rows.update(int(a) for a in perm[-32:] if a >= 0)            # the ragged last block
    return np.array(sorted(rows), dtype=np.int64)


@pytest.mark.parametrize("list_mode", ["tiles", "cluster", "atom"])
@pytest.mark.parametrize("precision", ["fp64", "mixed"])
def test_cfg1_full_parity(cfg1, precision, list_mode):
    import paper_2011_01207_b200 as pk
    s = cfg1
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_FP64 if precision == "fp64" else pk.TKHP_MIXED,
                                list_mode={"tiles": pk.TKHP_LIST_TILES, "cluster": pk.TKHP_LIST_CLUSTER, "atom": pk.TKHP_LIST_ATOM}[list_mode])
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    perm, pairs = P.nblist_view()
    oracle.check_perm(perm, s.pos, s.box)
    assert np.array_equal(pairs, oracle.block_pairs(perm, s.pos, s.box, s.cutoff + s.skin))
    tol = 1e-11 if precision == "fp64" else 1e-5
    E_ref = oracle.perm_field(s)                                  # full O(N^2): seconds
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    _assert_close(Eg.cpu().numpy(), E_ref, tol)
    rng = np.random.default_rng(1)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    _assert_close(P.tmatvec(mu).cpu().numpy(), oracle.tmatvec(s, mu), tol)
    # solve: oracle PCG to 1e-10, GPU tighter than the bar (Q11)
    mu_ref, _, _ = oracle.pcg_solve(s, E_ref, tol=1e-10)
    gtol = 1e-12 if precision == "fp64" else 1e-8
    mu_g, it, rms = P.polar_solve(Eg, tol=gtol)
    assert rms < gtol
    _assert_close(mu_g.cpu().numpy(), mu_ref, (1e-9 if precision == "fp64" else 1e-5))
    e_ref = oracle.polar_energy(mu_ref, E_ref)
    e_g = float(P.polar_energy(mu_g, Eg).cpu())
    assert abs(e_g - e_ref) <= (1e-9 if precision == "fp64" else 1e-6) * abs(e_ref)
    n_pair, _, _ = P.nblist_stats()
    assert n_pair == oracle.count_pairs(s)
    P.close()


@pytest.mark.parametrize("list_mode", ["tiles", "cluster", "atom"])
def test_cfg2_sampled_rows_mixed(cfg2, list_mode):
    """Config 2 (98,304 atoms, 15% solutes), MIXED: the configuration bench.py times."""
    import paper_2011_01207_b200 as pk
    s = cfg2
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED,
                                list_mode={"tiles": pk.TKHP_LIST_TILES, "cluster": pk.TKHP_LIST_CLUSTER, "atom": pk.TKHP_LIST_ATOM}[list_mode])
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    assert P.nblist_stats(count_pairs=False)[2] == {"tiles": pk.TKHP_LIST_TILES, "cluster": pk.TKHP_LIST_CLUSTER, "atom": pk.TKHP_LIST_ATOM}[list_mode]
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    perm, pairs = P.nblist_view()
    oracle.check_perm(perm, s.pos, s.box)
    assert np.array_equal(pairs, oracle.block_pairs(perm, s.pos, s.box, s.cutoff + s.skin))
    rows = _rows(s, perm)
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    E_rows = oracle.perm_field_rows(s, rows)
    _assert_close(Eg.cpu().numpy()[rows], E_rows, 1e-5)
    rng = np.random.default_rng(2)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    out = P.tmatvec(mu)
    _assert_close(out.cpu().numpy()[rows], oracle.tmatvec_rows(s, mu, rows), 1e-5)
    # properties that hold at any size: the solve's residual, recomputed with the oracle on rows
    mu_g, it, rms = P.polar_solve(Eg, tol=1e-8)
    assert rms < 1e-8 and it < 40
    mu_h = mu_g.cpu().numpy()
    res = Eg.cpu().numpy()[rows] - (mu_h[rows] / s.polarizability[rows, None]
                                    - oracle.tmatvec_rows(s, mu_h, rows))
    assert np.sqrt(np.mean(np.sum(res * res, axis=1))) < 5e-7     # FP32 pair math floor
    # energy equals -1/2 f mu.E evaluated on the host from the same arrays
    e_g = float(P.polar_energy(mu_g, Eg).cpu())
    assert abs(e_g - oracle.polar_energy(mu_h, Eg.cpu().numpy())) <= 1e-12 * abs(e_g)
    P.close()


@pytest.mark.parametrize("precision", ["mixed", "fp64"])
def test_groups_of_3_and_4_blocks_split_between_two_warps(precision):
    """A 48,000-atom box has 1,500 blocks in 444 groups of 3 or 4 blocks: every block is walked by two
    warps (even and odd list rows) whose parts are added in a fixed order.  Sampled
    rows against the oracle, the exact pair count, and bit-identical repeats."""
    import paper_2011_01207_b200 as pk
    from synth_inputs.generator import water_box
    s = water_box(16000, 78.3, 4801, solute_frac=0.1)
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_FP64 if precision == "fp64" else pk.TKHP_MIXED,
                                list_mode=pk.TKHP_LIST_ATOM)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    n_pair, n_slots, mode = P.nblist_stats()
    assert mode == pk.TKHP_LIST_ATOM and n_pair == oracle.count_pairs(s)
    perm, _ = P.nblist_view()
    n_blocks = perm.size // 32
    assert 3 <= n_blocks / 444 <= 4
    rows = _rows(s, perm, n_rand=768, n_blocks=6, seed=3)
    tol = 1e-11 if precision == "fp64" else 1e-5
    rng = np.random.default_rng(4)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    a = P.tmatvec(mu).cpu().numpy()
    _assert_close(a[rows], oracle.tmatvec_rows(s, mu, rows), tol)
    assert np.array_equal(a, P.tmatvec(mu).cpu().numpy())
    Eg = P.perm_field(s.charge, s.dipole, s.quad).cpu().numpy()
    _assert_close(Eg[rows], oracle.perm_field_rows(s, rows), tol)
    P.close()


# ----------------------------------------------------------------------------- config 2, every row
@pytest.fixture(scope="module")
def cfg2_oracle(cfg2):
    """The oracle on the whole of config 2, once for the module: field and one T.mu on all 98,304
    rows (about 10 s on 16 cores), and the PCG solve to 1e-10 (about a minute)."""
    s = cfg2
    rng = np.random.default_rng(2)
    probe = rng.standard_normal((s.n_atoms, 3)) * 0.1
    E = oracle.perm_field(s)
    T = oracle.tmatvec(s, probe)
    mu, it, rms = oracle.pcg_solve(s, E, tol=1e-10)
    assert rms < 1e-10
    return dict(probe=probe, E=E, T=T, mu=mu, e_pol=oracle.polar_energy(mu, E), n_pair=oracle.count_pairs(s))


@pytest.mark.parametrize("precision", ["mixed", "fp64"])
def test_cfg2_all_rows_and_solution_against_the_oracle(cfg2, cfg2_oracle, precision):
    """Config 2 (the system bench.py times), ATOM lists, BOTH precisions, EVERY row: field, T.mu, the
    induced dipoles and E_pol against the oracle (BASELINE.json: 1e-5 / 1e-11 rel-L2 for vectors,
    1e-5 for mu, 1e-6 for the energy), each with the per-row guard."""
    import paper_2011_01207_b200 as pk
    s, ref = cfg2, cfg2_oracle
    mixed = precision == "mixed"
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED if mixed else pk.TKHP_FP64, list_mode=pk.TKHP_LIST_ATOM)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    n_pair, n_slots, mode = P.nblist_stats()
    assert mode == pk.TKHP_LIST_ATOM and n_pair == ref["n_pair"]
    far, near, segs, far_on = P.nblist_atom_stats()
    assert far_on == mixed and far + near == n_slots and n_slots >= 2 * n_pair
    tol = 1e-5 if mixed else 1e-11
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    _assert_close(Eg.cpu().numpy(), ref["E"], tol)
    _assert_close(P.tmatvec(ref["probe"]).cpu().numpy(), ref["T"], tol)
    gtol = 1e-8 if mixed else 1e-12
    mu_g, it, rms = P.polar_solve(Eg, tol=gtol)
    assert rms < gtol
    # BASELINE.json's bar for mu is 1e-5 in both precisions; the FP64 run is held to what the oracle's
    # own stopping rule (rms 1e-10) leaves of its mu: a few 1e-9
    _assert_close(mu_g.cpu().numpy(), ref["mu"], 1e-5 if mixed else 1e-8)
    e_g = float(P.polar_energy(mu_g, Eg).cpu())
    assert abs(e_g - ref["e_pol"]) <= (1e-6 if mixed else 1e-9) * abs(ref["e_pol"])
    # the timing tolerance of bench.py: same iteration count as the oracle's PCG
    mu_t, it_t, rms_t = P.polar_solve(Eg, tol=1e-6)
    _, it_o, _ = oracle.pcg_solve(s, ref["E"], tol=1e-6)
    assert it_t == it_o and rms_t < 1e-6
    P.close()


# ----------------------------------------------------------------------------- config 3 (1,066,629 atoms)
def test_cfg3_sampled_rows_mixed():
    """BASELINE.json configs[3] (STMV-sized box), MIXED, ATOM lists: the bit-exact block-pair set
    (5.6e8 box tests in the oracle), the pair count against a k-d tree (scipy, periodic), 2,048 random
    rows + 8 whole blocks + the ragged last block of field and T.mu, and the solve's residual on
    those rows."""
    import paper_2011_01207_b200 as pk
    from scipy.spatial import cKDTree
    s = make_config(3)
    assert s.n_atoms == 1066629
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED, list_mode=pk.TKHP_LIST_ATOM)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    n_pair, n_slots, mode = P.nblist_stats()
    assert mode == pk.TKHP_LIST_ATOM
    perm, pairs = P.nblist_view()
    assert perm.size == 32 * 33333 and int((perm < 0).sum()) == 27          # phantoms pad the last block only
    oracle.check_perm(perm, s.pos, s.box)
    assert np.array_equal(pairs, oracle.block_pairs(perm, s.pos, s.box, s.cutoff + s.skin))
    # useful pairs: k-d tree count of ordered pairs incl. self within r_c (independent of both sides)
    w = oracle.wrap(s.pos, s.box)
    tree = cKDTree(w, boxsize=s.box)
    ordered_incl_self = int(tree.count_neighbors(tree, s.cutoff))
    assert n_pair == (ordered_incl_self - s.n_atoms) // 2
    assert 2 * n_pair <= n_slots <= 2.6 * n_pair
    rows = _rows(s, perm, n_rand=2048, n_blocks=8, seed=5)
    assert rows.size >= 2048 + 5
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    _assert_close(Eg.cpu().numpy()[rows], oracle.perm_field_rows(s, rows), 1e-5)
    rng = np.random.default_rng(6)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    out = P.tmatvec(mu).cpu().numpy()
    _assert_close(out[rows], oracle.tmatvec_rows(s, mu, rows), 1e-5)
    assert oracle.count_pairs_rows(s, rows) > 0
    mu_g, it, rms = P.polar_solve(Eg, tol=1e-8)
    assert rms < 1e-8 and it < 40
    mu_h = mu_g.cpu().numpy()
    res = Eg.cpu().numpy()[rows] - (mu_h[rows] / s.polarizability[rows, None] - oracle.tmatvec_rows(s, mu_h, rows))
    assert np.sqrt(np.mean(np.sum(res * res, axis=1))) < 5e-7
    e_g = float(P.polar_energy(mu_g, Eg).cpu())
    assert abs(e_g - oracle.polar_energy(mu_h, Eg.cpu().numpy())) <= 1e-12 * abs(e_g)
    P.close()


# ----------------------------------------------------------------------------- config 4: cutoff sweep
@pytest.mark.parametrize("precision", ["mixed", "fp64"])
@pytest.mark.parametrize("cutoff", [9.0, 12.0])
def test_cfg4_cutoff_sweep(cutoff, precision):
    """BASELINE.json configs[4]: the config-2 system at r_c = 9 and 12 A with beta = 3.8122 / r_c
    (Q9), both precisions, ATOM lists (list capacities and chunk counts no 7 A case
    reaches): field and T.mu on sampled rows, the solve's residual and iteration count."""
    import paper_2011_01207_b200 as pk
    s = make_config(4, cutoff=cutoff)
    assert abs(s.ewald_beta * cutoff - 0.5446 * 7.0) < 1e-12
    mixed = precision == "mixed"
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED if mixed else pk.TKHP_FP64, list_mode=pk.TKHP_LIST_ATOM)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    n_pair, n_slots, mode = P.nblist_stats()
    assert mode == pk.TKHP_LIST_ATOM
    from scipy.spatial import cKDTree
    tree = cKDTree(oracle.wrap(s.pos, s.box), boxsize=s.box)
    assert n_pair == (int(tree.count_neighbors(tree, s.cutoff)) - s.n_atoms) // 2
    assert 2 * n_pair <= n_slots <= 2.6 * n_pair
    perm, pairs = P.nblist_view()
    assert np.array_equal(pairs, oracle.block_pairs(perm, s.pos, s.box, s.cutoff + s.skin))
    rows = _rows(s, perm, n_rand=1024, n_blocks=4, seed=int(cutoff))
    tol = 1e-5 if mixed else 1e-11
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    _assert_close(Eg.cpu().numpy()[rows], oracle.perm_field_rows(s, rows), tol)
    rng = np.random.default_rng(8)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    _assert_close(P.tmatvec(mu).cpu().numpy()[rows], oracle.tmatvec_rows(s, mu, rows), tol)
    gtol = 1e-8 if mixed else 1e-12
    mu_g, it, rms = P.polar_solve(Eg, tol=gtol)
    assert rms < gtol and it < 40
    mu_h = mu_g.cpu().numpy()
    res = Eg.cpu().numpy()[rows] - (mu_h[rows] / s.polarizability[rows, None] - oracle.tmatvec_rows(s, mu_h, rows))
    assert np.sqrt(np.mean(np.sum(res * res, axis=1))) < (5e-7 if mixed else 1e-11)
    _, it6, rms6 = P.polar_solve(Eg, tol=1e-6)
    assert rms6 < 1e-6 and 6 <= it6 <= 14                      # 9-10 iterations at 9-12 A
    P.close()


_CFG4_ORACLE = {}


def _cfg4_oracle(cutoff):
    """Config 4's FP64 oracle solution at one cutoff (field on every row, PCG to 1e-10: 1-2 minutes of
    host time), computed once per cutoff for the four library variants below."""
    if cutoff not in _CFG4_ORACLE:
        s = make_config(4, cutoff=cutoff)
        E = oracle.perm_field(s)
        mu, _, rms = oracle.pcg_solve(s, E, tol=1e-10)
        assert rms < 1e-10
        _, it6, _ = oracle.pcg_solve(s, E, tol=1e-6)
        _CFG4_ORACLE[cutoff] = dict(s=s, E=E, mu=mu, e_pol=oracle.polar_energy(mu, E), it6=it6)
    return _CFG4_ORACLE[cutoff]


@pytest.mark.parametrize("variant", ["mixed", "fp64", "fixed", "stored_t"])
@pytest.mark.parametrize("cutoff", [9.0, 12.0])
def test_cfg4_solution_against_the_oracle(cutoff, variant):
    """BASELINE.json configs[4] asks for the "error versus the FP64 oracle": mu on EVERY row and E_pol against
    oracle.pcg_solve(tol=1e-10) at 9 and 12 A, at config 2's bars (MIXED 1e-5 / 1e-6, FP64 1e-8 / 1e-9), and the
    iteration count at 1e-6 against the oracle's.  TKHP_FIXED and TKHP_SOLVER_STORED_T run here on the paths
    no 7 A case reaches: several chunks per group, so one launch per product instead of the persistent kernel."""
    import paper_2011_01207_b200 as pk
    ref = _cfg4_oracle(cutoff)
    s = ref["s"]
    prec = {"mixed": pk.TKHP_MIXED, "fp64": pk.TKHP_FP64, "fixed": pk.TKHP_FIXED, "stored_t": pk.TKHP_MIXED}[variant]
    P = pk.Polarizer.for_system(s, precision=prec, list_mode=pk.TKHP_LIST_ATOM,
                                solver_flags=pk.TKHP_SOLVER_STORED_T if variant == "stored_t" else 0)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    assert P.nblist_stats(count_pairs=False)[2] == pk.TKHP_LIST_ATOM
    f64 = variant == "fp64"
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    _assert_close(Eg.cpu().numpy(), ref["E"], 1e-11 if f64 else 1e-5)
    mu_g, it, rms = P.polar_solve(Eg, tol=1e-12 if f64 else 1e-8)
    assert rms < (1e-12 if f64 else 1e-8)
    _assert_close(mu_g.cpu().numpy(), ref["mu"], 1e-8 if f64 else 1e-5)
    e_g = float(P.polar_energy(mu_g, Eg).cpu())
    assert abs(e_g - ref["e_pol"]) <= (1e-9 if f64 else 1e-6) * abs(ref["e_pol"])
    _, it6, rms6 = P.polar_solve(Eg, tol=1e-6)
    assert it6 == ref["it6"] and rms6 < 1e-6
    P.close()


def test_cfg2_fixed_point_mode(cfg2, cfg2_oracle):
    """Config 2 in the paper's FP mode (TKHP_FIXED): every row against the oracle at the
    MIXED bars, through the persistent solve kernel."""
    import paper_2011_01207_b200 as pk
    s, ref = cfg2, cfg2_oracle
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_FIXED, list_mode=pk.TKHP_LIST_ATOM)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    assert P.nblist_stats(count_pairs=False)[2] == pk.TKHP_LIST_ATOM
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    _assert_close(Eg.cpu().numpy(), ref["E"], 1e-5)
    _assert_close(P.tmatvec(ref["probe"]).cpu().numpy(), ref["T"], 1e-5)
    mu_g, it, rms = P.polar_solve(Eg, tol=1e-8)
    assert rms < 1e-8
    _assert_close(mu_g.cpu().numpy(), ref["mu"], 1e-5)
    e_g = float(P.polar_energy(mu_g, Eg).cpu())
    assert abs(e_g - ref["e_pol"]) <= 1e-6 * abs(ref["e_pol"])
    P.close()


def test_cfg2_stored_matrix_elements(cfg2, cfg2_oracle):
    """TKHP_SOLVER_STORED_T at the headline size: the product with stored elements on
    every row of config 2, and the solve that uses it (launch-per-matvec path), against the same oracle
    results, at the MIXED bars."""
    import paper_2011_01207_b200 as pk
    s, ref = cfg2, cfg2_oracle
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED, list_mode=pk.TKHP_LIST_ATOM,
                                solver_flags=pk.TKHP_SOLVER_STORED_T)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    n_pair, _, mode = P.nblist_stats()
    assert mode == pk.TKHP_LIST_ATOM and n_pair == ref["n_pair"]
    _assert_close(P.tmatvec(ref["probe"]).cpu().numpy(), ref["T"], 1e-5)
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    mu, _, rms = P.polar_solve(Eg, tol=1e-8)
    assert rms < 1e-8
    _assert_close(mu.cpu().numpy(), ref["mu"], 1e-5)
    e_g = float(P.polar_energy(mu, Eg).cpu())
    assert abs(e_g - ref["e_pol"]) <= 1e-6 * abs(ref["e_pol"])
    _, it6, rms6 = P.polar_solve(Eg, tol=1e-6)
    _, it_o, _ = oracle.pcg_solve(s, ref["E"], tol=1e-6)
    assert it6 == it_o and rms6 < 1e-6
    P.close()
