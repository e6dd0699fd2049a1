"""GPU parity: the CUDA library (through the C ABI binding) against the FP64 CPU oracle,
element by element on the same seeded inputs.  Tolerances are BASELINE.json's:
pair set bit-exact; field and T.mu rel-L2 <= 1e-5 (MIXED) / 1e-11 (FP64);
induced dipoles <= 1e-5 relative; energy <= 1e-6 relative."""
import numpy as np
import pytest

import oracle
from synth_inputs import make_config, tiny_cluster, water_box

pytestmark = pytest.mark.gpu

TOL_VEC = {"fp64": 1e-11, "mixed": 1e-5}


def _pk():
    import paper_2011_01207_b200 as pk
    return pk


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


def _polarizer(s, precision, list_mode="tiles"):
    pk = _pk()
    P = pk.Polarizer.for_system(
        s, precision=pk.TKHP_FP64 if precision == "fp64" else pk.TKHP_MIXED,
        list_mode={"tiles": pk.TKHP_LIST_TILES, "cluster": pk.TKHP_LIST_CLUSTER, "atom": pk.TKHP_LIST_ATOM}[list_mode])
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    return P


SYSTEMS = {
    "cfg0": lambda: make_config(0),
    "n2_open": lambda: tiny_cluster(2, 1, box=0.0, spread=2.0, group_size=1),
    "n3_open_onegroup": lambda: tiny_cluster(3, 2, box=0.0, spread=2.5, group_size=3),
    "n33_open": lambda: tiny_cluster(33, 3, box=0.0, spread=7.0, cutoff=5.0),
    "n65_periodic": lambda: tiny_cluster(65, 4, box=14.0, spread=14.0, cutoff=5.0, skin=1.0, ewald_beta=0.6),
    "n200_periodic_noewald": lambda: tiny_cluster(200, 5, box=20.0, spread=20.0, cutoff=6.0, skin=1.0),
    "water_1536_solutes": lambda: water_box(512, 24.85, 77, solute_frac=0.15),
    # large enough for the CLUSTER lists (box/2 > cutoff + group extent), small enough for Cholesky
    "water_6000": lambda: water_box(2000, 39.2, 78, solute_frac=0.1),
}


@pytest.fixture(scope="module", params=list(SYSTEMS))
def system(request):
    return SYSTEMS[request.param]()


# ------------------------------------------------------------------ neighbour list
def test_nblist_pair_set_is_bit_exact(system):
    s = system
    P = _polarizer(s, "mixed")
    perm, pairs = P.nblist_view()
    oracle.check_perm(perm, s.pos, s.box)                       # (N i, ii)
    want = oracle.block_pairs(perm, s.pos, s.box, s.cutoff + s.skin)   # (N iii)
    order = np.lexsort((pairs[:, 1], pairs[:, 0]))              # canonical sort
    assert np.array_equal(pairs[order], want)
    assert np.array_equal(order, np.arange(len(order))), "library list must already be sorted"
    n_pair, n_slots, mode = P.nblist_stats()
    assert n_pair == oracle.count_pairs(s)
    if s.n_atoms <= 2000:
        assert oracle.atom_pairs_covered(perm, pairs, s.pos, s.box, s.cutoff + s.skin)   # (N iv)
    P.close()


def test_nblist_is_deterministic_and_rebuildable():
    s = make_config(0)
    P = _polarizer(s, "mixed")
    perm1, pairs1 = P.nblist_view()
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    perm2, pairs2 = P.nblist_view()
    assert np.array_equal(perm1, perm2) and np.array_equal(pairs1, pairs2)
    # moved atoms -> different list on the same context
    P.nblist_build(s.pos + 0.37, s.polarizability, s.group_id)
    perm3, pairs3 = P.nblist_view()
    oracle.check_perm(perm3, s.pos + 0.37, s.box)
    assert np.array_equal(pairs3, oracle.block_pairs(perm3, s.pos + 0.37, s.box, s.cutoff + s.skin))
    P.close()


# ------------------------------------------------------------------ T.mu and field
@pytest.mark.parametrize("list_mode", ["tiles", "cluster", "atom"])
@pytest.mark.parametrize("precision", ["fp64", "mixed"])
def test_tmatvec_matches_oracle(system, precision, list_mode):
    s = system
    rng = np.random.default_rng(42)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    want = oracle.tmatvec(s, mu)
    P = _polarizer(s, precision, list_mode)
    got = P.tmatvec(mu).cpu().numpy()
    _assert_close(got, want, TOL_VEC[precision])
    P.close()


@pytest.mark.parametrize("list_mode", ["tiles", "cluster", "atom"])
@pytest.mark.parametrize("precision", ["fp64", "mixed"])
def test_perm_field_matches_oracle(system, precision, list_mode):
    s = system
    want = oracle.perm_field(s)
    P = _polarizer(s, precision, list_mode)
    got = P.perm_field(s.charge, s.dipole, s.quad).cpu().numpy()
    if np.linalg.norm(want) < 1e-12:      # isolated masked molecule: field is zero up to rounding
        assert np.abs(got).max() < 1e-12
    else:
        _assert_close(got, want, TOL_VEC[precision])
    P.close()


def test_cluster_mode_is_used_and_deterministic():
    """CLUSTER lists are active on a big enough box, fall back to TILES on a small one, and the
    cluster kernel (no atomics) returns bit-identical results run to run."""
    pk = _pk()
    s = SYSTEMS["water_6000"]()
    P = _polarizer(s, "mixed", "cluster")
    n_pair, n_slots, mode = P.nblist_stats()
    assert mode == pk.TKHP_LIST_CLUSTER and n_pair == oracle.count_pairs(s)
    assert 2 * n_pair <= n_slots <= 8 * n_pair          # ordered useful slots <= executed slots
    rng = np.random.default_rng(3)
    mu = rng.standard_normal((s.n_atoms, 3))
    a = P.tmatvec(mu).cpu().numpy()
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    b = P.tmatvec(mu).cpu().numpy()
    assert np.array_equal(a, b)
    P.close()
    small = _polarizer(make_config(0), "mixed", "cluster")
    assert small.nblist_stats()[2] == pk.TKHP_LIST_TILES
    small.close()


def test_atom_mode_lists_are_exact_and_deterministic():
    """ATOM lists: active on a big enough box, every list entry is a pair inside r_c (executed
    slots = ordered useful pairs + warp padding only), results bit-identical run to run, and the
    capacity fallback lands on CLUSTER with the same answers."""
    pk = _pk()
    s = SYSTEMS["water_6000"]()
    P = _polarizer(s, "mixed", "atom")
    n_pair, n_slots, mode = P.nblist_stats()
    assert mode == pk.TKHP_LIST_ATOM and n_pair == oracle.count_pairs(s)
    assert 2 * n_pair <= n_slots <= 3 * n_pair          # padding to the longest lane of a warp only
    rng = np.random.default_rng(3)
    mu = rng.standard_normal((s.n_atoms, 3))
    a = P.tmatvec(mu).cpu().numpy()
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    b = P.tmatvec(mu).cpu().numpy()
    assert np.array_equal(a, b)
    P.close()
    tight = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED, list_mode=pk.TKHP_LIST_ATOM,
                                    max_nbrs_per_atom=64)       # ~144 neighbours needed
    tight.nblist_build(s.pos, s.polarizability, s.group_id)
    assert tight.nblist_stats(count_pairs=False)[2] == pk.TKHP_LIST_CLUSTER
    c = tight.tmatvec(mu).cpu().numpy()
    assert _rel_l2(c, a) <= 1e-6
    tight.close()
    small = _polarizer(make_config(0), "mixed", "atom")
    assert small.nblist_stats()[2] == pk.TKHP_LIST_TILES
    small.close()


@pytest.mark.parametrize("precision", ["mixed", "fp64"])
@pytest.mark.parametrize("chunk", [256, 416])
def test_atom_mode_multi_chunk_staging(precision, chunk):
    """ATOM mode with a small shared-memory chunk: every group needs several interleaved chunks
    (DESIGN.md 5.3); T.mu and the field still match the oracle and the list is still exact."""
    pk = _pk()
    s = SYSTEMS["water_6000"]()
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_FP64 if precision == "fp64" else pk.TKHP_MIXED,
                                list_mode=pk.TKHP_LIST_ATOM, max_stage_per_chunk=chunk,
                                max_nbrs_per_atom=512)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    n_pair, n_slots, mode = P.nblist_stats()
    assert mode == pk.TKHP_LIST_ATOM and n_pair == oracle.count_pairs(s)
    assert 2 * n_pair <= n_slots <= 4 * n_pair
    rng = np.random.default_rng(5)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    _assert_close(P.tmatvec(mu).cpu().numpy(), oracle.tmatvec(s, mu), TOL_VEC[precision])
    E = P.perm_field(s.charge, s.dipole, s.quad).cpu().numpy()
    _assert_close(E, oracle.perm_field(s), TOL_VEC[precision])
    P.close()


def test_tmatvec_symmetry_on_gpu():
    """nu.T mu == mu.T nu for the GPU operator as well (FP64 mode)."""
    import torch
    s = make_config(0)
    P = _polarizer(s, "fp64")
    rng = np.random.default_rng(9)
    mu, nu = rng.standard_normal((2, s.n_atoms, 3))
    a = float((torch.as_tensor(nu, device="cuda") * P.tmatvec(mu)).sum())
    b = float((torch.as_tensor(mu, device="cuda") * P.tmatvec(nu)).sum())
    assert abs(a - b) <= 1e-12 * max(abs(a), abs(b))
    P.close()


# ------------------------------------------------------------------ solve and energy
@pytest.mark.parametrize("list_mode", ["tiles", "cluster", "atom"])
@pytest.mark.parametrize("precision", ["fp64", "mixed"])
@pytest.mark.parametrize("name", ["cfg0", "n65_periodic", "water_1536_solutes", "water_6000"])
def test_solve_and_energy_match_oracle(name, precision, list_mode):
    """Q11: both sides converge tighter than the parity bar so that truncation error does not
    mask arithmetic error (oracle: dense Cholesky; GPU: 1e-12 FP64 / 1e-8 MIXED)."""
    s = SYSTEMS[name]()
    E = oracle.perm_field(s)
    mu_ref = oracle.dense_solve(s, E)
    e_ref = oracle.polar_energy(mu_ref, E)
    P = _polarizer(s, precision, list_mode)
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    tol = 1e-12 if precision == "fp64" else 1e-8
    mu, it, rms = P.polar_solve(Eg, tol=tol, max_iter=100)
    assert rms < tol and 0 < it < 40
    mu_h = mu.cpu().numpy()
    _assert_close(mu_h, mu_ref, (1e-10 if precision == "fp64" else 1e-5))
    e_gpu = float(P.polar_energy(mu, Eg).cpu())
    assert abs(e_gpu - e_ref) <= (1e-10 if precision == "fp64" else 1e-6) * abs(e_ref)
    P.close()


def test_solve_iteration_counts_and_guess():
    s = make_config(0)
    P = _polarizer(s, "fp64")
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    E = Eg.cpu().numpy()
    for tol in (1e-5, 1e-6, 1e-8):
        _, it_ref, _ = oracle.pcg_solve(s, E, tol=tol)
        mu, it, rms = P.polar_solve(Eg, tol=tol)
        assert it == it_ref and rms < tol
    mu2, it2, rms2 = P.polar_solve(Eg, tol=1e-8, guess=mu)
    assert it2 == 0
    pk = _pk()
    with pytest.raises(pk.TkhpError) as e:
        P.polar_solve(Eg, tol=1e-30, max_iter=2)
    assert e.value.code == -5
    P.close()


def test_two_site_closed_form_through_the_library(golden):
    """Pin P8 through the GPU path (open boundary, beta = 0)."""
    import torch
    from synth_inputs import System
    g = golden["P8_two_site"]
    s = System(name="two", box=0.0, pos=np.array([[0, 0, 0], [0, 0, g["R"]]], float),
               charge=np.zeros(2), dipole=np.zeros((2, 3)), quad=np.zeros((2, 6)),
               polarizability=np.array(g["alpha"]), group_id=np.array([0, 1], np.int32),
               cutoff=7.0, skin=2.0, ewald_beta=0.0, thole_a=g["a"])
    P = _polarizer(s, "fp64")
    for axis, key in ((2, "par"), (0, "perp")):
        E = np.zeros((2, 3)); E[:, axis] = g["E"]
        mu, it, rms = P.polar_solve(E, tol=1e-14)
        np.testing.assert_allclose(mu.cpu().numpy()[:, axis], g["mu_" + key], rtol=1e-12)
        e = float(P.polar_energy(mu, torch.as_tensor(E, device="cuda")).cpu())
        assert e == pytest.approx(g["Epol_" + key], rel=1e-12)
    P.close()


# ------------------------------------------------------------------ host entry and errors
def test_polarize_host_matches_device_calls():
    pk = _pk()
    s = make_config(0)
    P = _polarizer(s, "mixed")
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    mu, it, rms = P.polar_solve(Eg, tol=1e-6)
    e = float(P.polar_energy(mu, Eg).cpu())
    h_mu = np.zeros((s.n_atoms, 3)); h_E = np.zeros((s.n_atoms, 3)); h_e = np.zeros(1)
    it2, rms2, ok = pk.tkhp_polarize_host(P.ctx, s.pos, s.polarizability, s.group_id, s.charge,
                                          s.dipole, s.quad, 1e-6, 100, h_mu, h_E, h_e)
    assert ok and it2 == it
    np.testing.assert_allclose(h_E, Eg.cpu().numpy(), rtol=0, atol=1e-9)
    assert _rel_l2(h_mu, mu.cpu().numpy()) < 1e-6
    assert abs(h_e[0] - e) < 1e-6 * abs(e)
    P.close()


def test_error_paths_on_device():
    pk = _pk()
    s = make_config(0)
    P = pk.Polarizer.for_system(s)
    with pytest.raises(pk.TkhpError) as e:
        P.tmatvec(np.zeros((s.n_atoms, 3)))
    assert e.value.code == -4                       # TKHP_ENOLIST
    bad = s.pos.copy(); bad[5, 1] = np.nan
    P.nblist_build(bad, s.polarizability, s.group_id)
    with pytest.raises(pk.TkhpError) as e:
        P.nblist_view()
    assert e.value.code == -7                       # TKHP_ENONFINITE
    al = s.polarizability.copy(); al[7] = 0.0
    P.nblist_build(s.pos, al, s.group_id)
    with pytest.raises(pk.TkhpError) as e:
        P.tmatvec(np.zeros((s.n_atoms, 3)))
    assert e.value.code == -7
    P.nblist_build(s.pos, s.polarizability, s.group_id)   # context recovers
    P.tmatvec(np.ones((s.n_atoms, 3)))
    P.close()
    tiny = pk.Polarizer.for_system(s, max_tiles_per_block=1)
    tiny.nblist_build(s.pos, s.polarizability, s.group_id)
    with pytest.raises(pk.TkhpError) as e:
        tiny.nblist_view()
    assert e.value.code == -6                       # TKHP_ECAPACITY
    tiny.close()


# ------------------------------------------------------------------ solver paths, streams, open boundary
@pytest.mark.parametrize("flags", ["persistent", "no_persistent", "no_fused_step"])
def test_every_solver_path_agrees_with_the_oracle(flags):
    """tkhp_polar_solve has three paths in MIXED/ATOM mode: the persistent cooperative kernel, the
    launch-per-matvec loop with the fused update+direction kernel, and the same with two kernels
    (tkhp_params.solver_flags forces the fall-backs).  Each against the dense Cholesky solution, with
    the oracle's iteration count."""
    pk = _pk()
    s = SYSTEMS["water_6000"]()
    f = {"persistent": 0, "no_persistent": pk.TKHP_SOLVER_NO_PERSISTENT,
         "no_fused_step": pk.TKHP_SOLVER_NO_PERSISTENT | pk.TKHP_SOLVER_NO_FUSED_STEP}[flags]
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED, list_mode=pk.TKHP_LIST_ATOM, solver_flags=f)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    assert P.nblist_stats(count_pairs=False)[2] == pk.TKHP_LIST_ATOM
    E_ref = oracle.perm_field(s)
    mu_ref = oracle.dense_solve(s, E_ref)
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    mu, it, rms = P.polar_solve(Eg, tol=1e-8)
    assert rms < 1e-8
    _assert_close(mu.cpu().numpy(), mu_ref, 1e-5)
    for tol in (1e-5, 1e-6):
        _, it_ref, _ = oracle.pcg_solve(s, E_ref, tol=tol)
        mu_t, it_t, rms_t = P.polar_solve(Eg, tol=tol)
        assert it_t == it_ref and rms_t < tol
    # bit-reproducible, and a converged guess needs no iteration
    mu_b, it_b, _ = P.polar_solve(Eg, tol=1e-8)
    assert it_b == it and np.array_equal(mu_b.cpu().numpy(), mu.cpu().numpy())
    _, it0, _ = P.polar_solve(Eg, tol=1e-6, guess=mu)
    assert it0 == 0
    with pytest.raises(pk.TkhpError) as e:
        P.polar_solve(Eg, tol=1e-30, max_iter=2)
    assert e.value.code == -5                       # TKHP_ENOCONV
    P.close()


@pytest.mark.parametrize("kernel", ["k_pcg_persist", "k_pcg_tiles"])
def test_broken_grid_barrier_falls_back_to_launch_per_matvec(kernel):
    """A persistent solve kernel whose grid barrier breaks (here: TKHP_SOLVER_TEST_BARRIER_FAULT makes
    the last CTA leave before its first arrival; the others give up after 2 s of %globaltimer) writes
    nothing to d_mu.  tkhp_polar_solve then repeats the solve with one launch per product:
    same answer and iteration count as a context that never used the persistent kernel, the guess is
    honoured, the event is counted once, and later solves stay on the fall-back path (no second wait)."""
    import time
    import torch
    pk = _pk()
    s, mode = (SYSTEMS["water_6000"](), pk.TKHP_LIST_ATOM) if kernel == "k_pcg_persist" else (SYSTEMS["cfg0"](), pk.TKHP_LIST_TILES)
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED, list_mode=mode, solver_flags=pk.TKHP_SOLVER_TEST_BARRIER_FAULT)
    Q = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED, list_mode=mode, solver_flags=pk.TKHP_SOLVER_NO_PERSISTENT)
    for X in (P, Q):
        X.nblist_build(s.pos, s.polarizability, s.group_id)
    assert P.nblist_stats(count_pairs=False)[2] == mode
    Eg = Q.perm_field(s.charge, s.dipole, s.quad)
    mu_q, it_q, rms_q = Q.polar_solve(Eg, tol=1e-7)
    # a guess that is nowhere near alpha E: were it overwritten or ignored, the iteration count would differ
    guess = mu_q * 0.5
    mu_qg, it_qg, _ = Q.polar_solve(Eg, tol=1e-7, guess=guess)
    assert pk.tkhp_profile_read_build(P.ctx)["barrier_timeouts"] == 0
    t0 = time.perf_counter()
    mu_p, it_p, rms_p = P.polar_solve(Eg, tol=1e-7, guess=guess)
    waited = time.perf_counter() - t0
    assert 1.9 < waited < 30.0, waited                       # the barrier's time bound is a time, not a poll count
    assert pk.tkhp_profile_read_build(P.ctx)["barrier_timeouts"] == 1
    assert it_p == it_qg and rms_p < 1e-7
    # ATOM lists: one writer per atom, bit-reproducible; TILES: FP64 atomics, order-dependent last bits
    same = (lambda a, b: np.array_equal(a, b)) if kernel == "k_pcg_persist" else (lambda a, b: _rel_l2(a, b) < 1e-9)
    assert same(mu_p.cpu().numpy(), mu_qg.cpu().numpy())
    _assert_close(mu_p.cpu().numpy(), oracle.dense_solve(s, oracle.perm_field(s)), 1e-5)
    t0 = time.perf_counter()
    mu_2, it_2, _ = P.polar_solve(Eg, tol=1e-7)
    torch.cuda.synchronize()
    assert time.perf_counter() - t0 < 1.0
    assert it_2 == it_q and same(mu_2.cpu().numpy(), mu_q.cpu().numpy())
    assert pk.tkhp_profile_read_build(P.ctx)["barrier_timeouts"] == 1
    P.close(); Q.close()


def test_own_stream_replays_the_build_as_a_graph():
    """On a stream of the caller's (not the legacy default stream) the list build is captured once
    and replayed as a CUDA graph: same lists, same results, also after the inputs change in place
    and after other input tensors are passed."""
    import torch
    pk = _pk()
    s = SYSTEMS["water_6000"]()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        P = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED, list_mode=pk.TKHP_LIST_ATOM)
        d_pos = torch.as_tensor(s.pos, device="cuda")
        d_al = torch.as_tensor(s.polarizability, device="cuda")
        d_g = torch.as_tensor(s.group_id, dtype=torch.int32, device="cuda")
        for rep in range(3):                         # capture, then two replays
            pk.tkhp_nblist_build(P.ctx, d_pos, d_al, d_g, st)
            perm, pairs = P.nblist_view(st)
            oracle.check_perm(perm, s.pos, s.box)
            assert np.array_equal(pairs, oracle.block_pairs(perm, s.pos, s.box, s.cutoff + s.skin))
        rng = np.random.default_rng(9)
        mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
        _assert_close(P.tmatvec(mu, stream=st).cpu().numpy(), oracle.tmatvec(s, mu), 1e-5)
        # same buffers, new positions: the replayed graph reads the new contents
        moved = s.pos + np.array([0.31, -0.17, 0.23])
        d_pos.copy_(torch.as_tensor(moved, device="cuda"))
        pk.tkhp_nblist_build(P.ctx, d_pos, d_al, d_g, st)
        perm, pairs = P.nblist_view(st)
        oracle.check_perm(perm, moved, s.box)
        assert np.array_equal(pairs, oracle.block_pairs(perm, moved, s.box, s.cutoff + s.skin))
        # other buffers: re-captured
        d_pos2 = torch.as_tensor(s.pos, device="cuda")
        pk.tkhp_nblist_build(P.ctx, d_pos2, d_al, d_g, st)
        perm, pairs = P.nblist_view(st)
        oracle.check_perm(perm, s.pos, s.box)
        _assert_close(P.tmatvec(mu, stream=st).cpu().numpy(), oracle.tmatvec(s, mu), 1e-5)
        # an integrator that alternates between position buffers: both graphs stay cached,
        # every build is a replay, and each replay reads the buffer it was captured with
        base = pk.tkhp_profile_read_build(P.ctx)
        assert base == dict(graph_captures=2, graph_replays=5, plain_builds=0, graphs_off=False, barrier_timeouts=0)
        for rep in range(6):
            buf, want = (d_pos, moved) if rep % 2 == 0 else (d_pos2, s.pos)
            pk.tkhp_nblist_build(P.ctx, buf, d_al, d_g, st)
            if rep >= 4:
                perm, pairs = P.nblist_view(st)
                oracle.check_perm(perm, want, s.box)
                assert np.array_equal(pairs, oracle.block_pairs(perm, want, s.box, s.cutoff + s.skin))
        now = pk.tkhp_profile_read_build(P.ctx)
        assert now == dict(graph_captures=2, graph_replays=11, plain_builds=0, graphs_off=False, barrier_timeouts=0)
        # more pointer triples than slots: the least recently used graph is replaced, results stay right
        extra = [torch.as_tensor(s.pos, device="cuda") for _ in range(4)]
        for buf in extra:
            pk.tkhp_nblist_build(P.ctx, buf, d_al, d_g, st)
        pk.tkhp_nblist_build(P.ctx, d_pos, d_al, d_g, st)          # evicted by now: captured again
        perm, pairs = P.nblist_view(st)
        oracle.check_perm(perm, moved, s.box)
        assert np.array_equal(pairs, oracle.block_pairs(perm, moved, s.box, s.cutoff + s.skin))
        assert pk.tkhp_profile_read_build(P.ctx) == dict(graph_captures=7, graph_replays=16, plain_builds=0,
                                                         graphs_off=False, barrier_timeouts=0)
        # the legacy default stream cannot be captured: plain launches, counted as such
        torch.cuda.synchronize()
        pk.tkhp_nblist_build(P.ctx, d_pos2, d_al, d_g, 0)
        perm, pairs = P.nblist_view(0)
        oracle.check_perm(perm, s.pos, s.box)
        assert pk.tkhp_profile_read_build(P.ctx)["plain_builds"] == 1
        _assert_close(P.tmatvec(mu, stream=st).cpu().numpy(), oracle.tmatvec(s, mu), 1e-5)
        P.close()


def test_open_boundary_elongated_system():
    """An open-boundary system much wider than the cell table's finest grid: the sort
    grid is clamped to 2^6 cells per axis, the build does not fail, and list
    and results still match the oracle."""
    pk = _pk()
    s = tiny_cluster(300, 21, box=0.0, spread=9.0, cutoff=6.0, skin=1.0)
    pos = s.pos.copy()
    pos[:, 0] *= 60.0                                # 540 A long, 9 A across
    s = s.with_(pos=pos)
    for precision in ("fp64", "mixed"):
        P = _polarizer(s, precision, "atom")
        perm, pairs = P.nblist_view()
        oracle.check_perm(perm, s.pos, s.box)
        assert np.array_equal(pairs, oracle.block_pairs(perm, s.pos, s.box, s.cutoff + s.skin))
        assert P.nblist_stats()[0] == oracle.count_pairs(s)
        _assert_close(P.perm_field(s.charge, s.dipole, s.quad).cpu().numpy(), oracle.perm_field(s), TOL_VEC[precision])
        P.close()


# ------------------------------------------------------------------ TKHP_FIXED: the paper's FP mode
@pytest.mark.parametrize("list_mode", ["tiles", "cluster", "atom"])
@pytest.mark.parametrize("name", ["cfg0", "water_6000"])
def test_fixed_point_mode_matches_the_oracle(name, list_mode):
    """TKHP_FIXED (eqs 2-3): FP32 pair math, int64 containers with 34 fractional bits for the
    field and T.mu accumulators and 30 for the energy.  Same bars as MIXED (BASELINE.json), bit-identical
    repeats (in TILES mode too, where the containers are filled by integer atomics in any order), and the
    energy is an integer multiple of 2^-30 kcal/mol."""
    pk = _pk()
    s = SYSTEMS[name]()
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_FIXED,
                                list_mode={"tiles": pk.TKHP_LIST_TILES, "cluster": pk.TKHP_LIST_CLUSTER, "atom": pk.TKHP_LIST_ATOM}[list_mode])
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    E_ref = oracle.perm_field(s)
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    _assert_close(Eg.cpu().numpy(), E_ref, 1e-5)
    rng = np.random.default_rng(12)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    t1 = P.tmatvec(mu).cpu().numpy()
    _assert_close(t1, oracle.tmatvec(s, mu), 1e-5)
    for _ in range(3):
        assert np.array_equal(P.tmatvec(mu).cpu().numpy(), t1)
        assert np.array_equal(P.perm_field(s.charge, s.dipole, s.quad).cpu().numpy(), Eg.cpu().numpy())
    mu_ref = oracle.dense_solve(s, E_ref)
    mu_g, it, rms = P.polar_solve(Eg, tol=1e-8)
    assert rms < 1e-8
    _assert_close(mu_g.cpu().numpy(), mu_ref, 1e-5)
    e_ref = oracle.polar_energy(mu_ref, E_ref)
    e_g = float(P.polar_energy(mu_g, Eg).cpu())
    assert abs(e_g - e_ref) <= 1e-6 * abs(e_ref)
    scaled = e_g * float(1 << oracle.FIX_ENERGY_BITS)
    assert scaled == np.rint(scaled) and int(oracle.to_fixed(e_g, oracle.FIX_ENERGY_BITS)) == int(scaled)
    # one conversion per atom (Q21): from the same arrays the oracle's fixed-point energy is the same integer
    assert e_g == oracle.polar_energy_fixed(mu_g.cpu().numpy(), Eg.cpu().numpy())
    P.close()


@pytest.mark.parametrize("list_mode", ["tiles", "atom"])
def test_fixed_point_accumulators_hold_multiples_of_2_to_minus_34(list_mode):
    """Open boundary, beta = 0 (no self term), one atom per group (no mask correction): the library's
    T.mu output IS the accumulator, so every component must be an integer multiple of 2^-34 (eq. 3)."""
    pk = _pk()
    s = tiny_cluster(200, 31, box=0.0, spread=14.0, group_size=1, cutoff=6.0, skin=1.0)
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_FIXED,
                                list_mode=pk.TKHP_LIST_TILES if list_mode == "tiles" else pk.TKHP_LIST_ATOM)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    rng = np.random.default_rng(13)
    mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
    out = P.tmatvec(mu).cpu().numpy()
    _assert_close(out, oracle.tmatvec(s, mu), 1e-5)
    a = oracle.to_fixed(out, oracle.FIX_VEC_BITS)
    assert np.array_equal(oracle.from_fixed(a, oracle.FIX_VEC_BITS), out)
    assert np.abs(out).max() > 1e-3                              # (not trivially zero)
    # MIXED on the same system is NOT confined to that grid
    Pm = pk.Polarizer.for_system(s, precision=pk.TKHP_MIXED,
                                 list_mode=pk.TKHP_LIST_TILES if list_mode == "tiles" else pk.TKHP_LIST_ATOM)
    Pm.nblist_build(s.pos, s.polarizability, s.group_id)
    om = Pm.tmatvec(mu).cpu().numpy()
    assert not np.array_equal(oracle.from_fixed(oracle.to_fixed(om, oracle.FIX_VEC_BITS), oracle.FIX_VEC_BITS), om)
    P.close(); Pm.close()


# ------------------------------------------------------------------ stored real-space matrix elements
@pytest.mark.parametrize("variant", ["mixed", "fixed", "multi_chunk", "no_ewald"])
def test_stored_matrix_elements_match_the_oracle(variant):
    """TKHP_SOLVER_STORED_T ("precompute the real space matrix elements before the
    iterations"): the two radial factors of every list slot are computed once after a build and every
    T.mu product streams them.  Products, the PCG solve (iteration counts included) and the energy
    against the oracle; a second build with moved atoms must replace the stored elements."""
    pk = _pk()
    if variant == "no_ewald":
        s = tiny_cluster(200, 31, box=0.0, spread=14.0, group_size=1, cutoff=6.0, skin=1.0)   # open boundary, beta = 0: no far class
        kw = {}
    else:
        s = SYSTEMS["water_6000"]()
        kw = {"max_stage_per_chunk": 416, "max_nbrs_per_atom": 512} if variant == "multi_chunk" else {}
    P = pk.Polarizer.for_system(s, precision=pk.TKHP_FIXED if variant == "fixed" else pk.TKHP_MIXED,
                                list_mode=pk.TKHP_LIST_ATOM, solver_flags=pk.TKHP_SOLVER_STORED_T, **kw)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    n_pair, _, mode = P.nblist_stats()
    assert mode == pk.TKHP_LIST_ATOM and n_pair == oracle.count_pairs(s)
    rng = np.random.default_rng(21)
    for rep in range(2):                                   # the second product re-uses the stored elements
        mu = rng.standard_normal((s.n_atoms, 3)) * 0.1
        _assert_close(P.tmatvec(mu).cpu().numpy(), oracle.tmatvec(s, mu), 1e-5)
    a, b = P.tmatvec(mu).cpu().numpy(), P.tmatvec(mu).cpu().numpy()
    assert np.array_equal(a, b)                            # bit-reproducible
    # solve and energy through the launch-per-matvec path with stored products
    E_ref = oracle.perm_field(s)
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    mu_ref, _, _ = oracle.pcg_solve(s, E_ref, tol=1e-10)
    mu_g, it, rms = P.polar_solve(Eg, tol=1e-8)
    assert rms < 1e-8
    _assert_close(mu_g.cpu().numpy(), mu_ref, 1e-5)
    e_ref = oracle.polar_energy(mu_ref, E_ref)
    assert abs(float(P.polar_energy(mu_g, Eg).cpu()) - e_ref) <= 1e-6 * abs(e_ref)
    for tol in (1e-5, 1e-6):
        _, it_ref, _ = oracle.pcg_solve(s, E_ref, tol=tol)
        _, it_t, rms_t = P.polar_solve(Eg, tol=tol)
        assert it_t == it_ref and rms_t < tol
    # a new list (atoms moved by up to 0.3 A) must not see the old elements
    import copy
    s2 = copy.copy(s)
    s2.pos = s.pos + np.random.default_rng(3).uniform(-0.3, 0.3, size=s.pos.shape)
    P.nblist_build(s2.pos, s2.polarizability, s2.group_id)
    _assert_close(P.tmatvec(mu).cpu().numpy(), oracle.tmatvec(s2, mu), 1e-5)
    P.close()


def test_stored_matrix_elements_flag_is_ignored_in_fp64():
    """The flag only changes MIXED/FIXED ATOM-mode contexts; in FP64 it is accepted and ignored (no
    extra workspace), so that one parameter set can serve both precisions."""
    pk = _pk()
    s = SYSTEMS["water_1536_solutes"]()
    P0 = pk.Polarizer.for_system(s, precision=pk.TKHP_FP64, list_mode=pk.TKHP_LIST_ATOM)
    P1 = pk.Polarizer.for_system(s, precision=pk.TKHP_FP64, list_mode=pk.TKHP_LIST_ATOM,
                                 solver_flags=pk.TKHP_SOLVER_STORED_T)
    assert P0.workspace.numel() == P1.workspace.numel()
    P1.nblist_build(s.pos, s.polarizability, s.group_id)
    mu = np.random.default_rng(2).standard_normal((s.n_atoms, 3)) * 0.1
    _assert_close(P1.tmatvec(mu).cpu().numpy(), oracle.tmatvec(s, mu), 1e-11)
    P0.close(); P1.close()


@pytest.mark.parametrize("precision", ["mixed", "fp64", "fixed"])
@pytest.mark.parametrize("flags", ["persistent", "no_persistent"])
def test_tiles_mode_solver_paths(flags, precision):
    """Config 0 (box too small for the finer lists: TILES): the persistent cooperative solve kernel
    (k_pcg_tiles) and the launch-per-matvec loop against the dense solution, with the oracle's
    iteration counts, a converged guess and open-boundary input."""
    pk = _pk()
    s = SYSTEMS["cfg0"]()
    prec = {"mixed": pk.TKHP_MIXED, "fp64": pk.TKHP_FP64, "fixed": pk.TKHP_FIXED}[precision]
    P = pk.Polarizer.for_system(s, precision=prec, list_mode=pk.TKHP_LIST_ATOM,
                                solver_flags=0 if flags == "persistent" else pk.TKHP_SOLVER_NO_PERSISTENT)
    P.nblist_build(s.pos, s.polarizability, s.group_id)
    assert P.nblist_stats(count_pairs=False)[2] == pk.TKHP_LIST_TILES
    E_ref = oracle.perm_field(s)
    mu_ref = oracle.dense_solve(s, E_ref)
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    tight = 1e-12 if precision == "fp64" else 1e-8
    mu, it, rms = P.polar_solve(Eg, tol=tight)
    assert rms < tight
    _assert_close(mu.cpu().numpy(), mu_ref, 1e-10 if precision == "fp64" else 1e-5)
    for tol in (1e-5, 1e-6):
        _, it_ref, _ = oracle.pcg_solve(s, E_ref, tol=tol)
        _, it_t, rms_t = P.polar_solve(Eg, tol=tol)
        assert it_t == it_ref and rms_t < tol
    _, it0, _ = P.polar_solve(Eg, tol=1e-6, guess=mu)
    assert it0 == 0
    e_ref = oracle.polar_energy(mu_ref, E_ref)
    assert abs(float(P.polar_energy(mu, Eg).cpu()) - e_ref) <= 1e-6 * abs(e_ref)
    P.close()
    # open boundary, no Ewald: 200 random sites
    s2 = tiny_cluster(200, 31, box=0.0, spread=14.0, group_size=1, cutoff=6.0, skin=1.0)
    P2 = pk.Polarizer.for_system(s2, precision=prec, list_mode=pk.TKHP_LIST_TILES,
                                 solver_flags=0 if flags == "persistent" else pk.TKHP_SOLVER_NO_PERSISTENT)
    P2.nblist_build(s2.pos, s2.polarizability, s2.group_id)
    E2 = oracle.perm_field(s2)
    mu2, _, _ = P2.polar_solve(P2.perm_field(s2.charge, s2.dipole, s2.quad), tol=tight)
    _assert_close(mu2.cpu().numpy(), oracle.dense_solve(s2, E2), 1e-10 if precision == "fp64" else 1e-5)
    P2.close()
