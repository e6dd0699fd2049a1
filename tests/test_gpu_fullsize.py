"""GPU parity at BASELINE.json's full sizes (configs 1 and 2), in the launch configuration
bench.py times: sampled rows the oracle computes one by one, the bit-exact block-pair set,
the useful-pair count, and properties that hold at any size."""
import numpy as np
import pytest

import oracle
from synth_inputs import make_config

pytestmark = pytest.mark.gpu


def _rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(b))


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
    assert _rel_l2(Eg.cpu().numpy(), E_ref) <= tol
    rng = np.random.default_rng(1)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    assert _rel_l2(P.tmatvec(mu).cpu().numpy(), oracle.tmatvec(s, mu)) <= tol
    # solve: oracle PCG to 1e-10, GPU tighter than the bar (Q11)
    mu_ref, _, _ = oracle.pcg_solve(s, E_ref, tol=1e-10)
    gtol = 1e-12 if precision == "fp64" else 1e-8
    mu_g, it, rms = P.polar_solve(Eg, tol=gtol)
    assert rms < gtol
    assert _rel_l2(mu_g.cpu().numpy(), mu_ref) <= (1e-9 if precision == "fp64" else 1e-5)
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
    assert _rel_l2(Eg.cpu().numpy()[rows], E_rows) <= 1e-5
    rng = np.random.default_rng(2)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    out = P.tmatvec(mu)
    assert _rel_l2(out.cpu().numpy()[rows], oracle.tmatvec_rows(s, mu, rows)) <= 1e-5
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
    assert _rel_l2(a[rows], oracle.tmatvec_rows(s, mu, rows)) <= tol
    assert np.array_equal(a, P.tmatvec(mu).cpu().numpy())
    Eg = P.perm_field(s.charge, s.dipole, s.quad).cpu().numpy()
    assert _rel_l2(Eg[rows], oracle.perm_field_rows(s, rows)) <= tol
    P.close()
