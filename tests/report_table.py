"""Result table of BASELINE.md section 3 (SURVEY 8(d) protocol), written as markdown rows.

    python tests/report_table.py [--configs 0,1,2,3] [--sweep] > gpurun_out/table.md

Not a test (pytest does not collect it): it needs a B200 and several minutes of host time for the
O(N^2) oracle.  Per config and precision: pair counts, slots evaluated, list build / field /
matvec / solve times (CUDA events inside the library, median of --reps), the live pair-kernel
durations, PCG iterations at tol 1e-6, and the errors against the FP64 oracle (full system up to
config 2, seeded random rows plus whole blocks on config 3).  --sweep adds config 4 (the config-2
system at r_c = 7, 9, 12 A, beta = 3.8122 / r_c) in both precisions.
It lives under tests/ because it calls the oracle, which only tests, smoke() and bench.py may do.
"""
from __future__ import annotations

import argparse
import statistics
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import oracle  # noqa: E402
from synth_inputs import make_config  # noqa: E402


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(b))


def sample_rows(s, perm, n_rand, n_blocks, seed=0):
    rng = np.random.default_rng(seed)
    rows = set(rng.choice(s.n_atoms, size=min(n_rand, s.n_atoms), replace=False).tolist())
    nb = perm.size // 32
    for b in rng.choice(nb, size=min(n_blocks, nb), replace=False):
        rows.update(int(a) for a in perm[32 * b:32 * b + 32] if a >= 0)
    rows.update(int(a) for a in perm[-32:] if a >= 0)
    return np.array(sorted(rows), dtype=np.int64)


def run_one(s, label, precision, reps, full_oracle):
    import torch
    import paper_2011_01207_b200 as pk
    prec = pk.TKHP_FP64 if precision == "fp64" else pk.TKHP_MIXED
    P = pk.Polarizer.for_system(s, precision=prec, list_mode=pk.TKHP_LIST_ATOM)
    rng = np.random.default_rng(1)
    probe = rng.standard_normal((s.n_atoms, 3)) * 0.1
    t = dict(build=[], field=[], solve=[], energy=[], tmu=[], fld=[])
    it = 0
    for r in range(reps + 2):
        pk.tkhp_profile_reset(P.ctx, True)
        P.nblist_build(s.pos, s.polarizability, s.group_id)
        E = P.perm_field(s.charge, s.dipole, s.quad)
        mu, it, rms = P.polar_solve(E, tol=1e-6)
        e_pol = float(P.polar_energy(mu, E).cpu())
        torch.cuda.synchronize()
        if r < 2:
            continue
        ph = P.timings()
        pr = pk.tkhp_profile_read(P.ctx)
        for k in ("build", "field", "solve", "energy"):
            t[k].append(ph[k])
        t["tmu"].append(pr["tmatvec_ms"] / max(pr["n_tmatvec"], 1))
        t["fld"].append(pr["field_ms"] / max(pr["n_field"], 1))
    med = {k: statistics.median(v) for k, v in t.items()}
    n_pair, n_slots, mode = P.nblist_stats()
    perm, _ = P.nblist_view()
    # ---- errors against the oracle
    t0 = time.perf_counter()
    Eg = P.perm_field(s.charge, s.dipole, s.quad)
    Tg = P.tmatvec(probe).cpu().numpy()
    gtol = 1e-12 if precision == "fp64" else 1e-8
    mu_g, _, _ = P.polar_solve(Eg, tol=gtol)
    e_g = float(P.polar_energy(mu_g, Eg).cpu())
    if full_oracle:
        E_ref = oracle.perm_field(s)
        T_ref = oracle.tmatvec(s, probe)
        mu_ref, _, _ = oracle.pcg_solve(s, E_ref, tol=1e-10)
        e_ref = oracle.polar_energy(mu_ref, E_ref)
        errs = (rel_l2(Tg, T_ref), rel_l2(Eg.cpu().numpy(), E_ref), rel_l2(mu_g.cpu().numpy(), mu_ref),
                abs(e_g - e_ref) / abs(e_ref))
        err_txt = "%.1e / %.1e / %.1e, %.1e" % errs
    else:
        rows = sample_rows(s, perm, 2048, 8)
        E_rows = oracle.perm_field_rows(s, rows)
        T_rows = oracle.tmatvec_rows(s, probe, rows)
        err_txt = "%.1e / %.1e / -, - (%d sampled rows)" % (rel_l2(Tg[rows], T_rows),
                                                           rel_l2(Eg.cpu().numpy()[rows], E_rows), rows.size)
    oracle_s = time.perf_counter() - t0
    P.close()
    gp = lambda ms: n_pair / (ms * 1e-3) / 1e9
    print("| %s | %s | %d | %d | %d | %.3f | %.4f (%.0f) | %.4f (%.0f) | %d | %.3f | %s | %.0f (%d) |" % (
        label, precision, s.n_atoms, n_pair, n_slots, med["build"], med["fld"], gp(med["fld"]), med["tmu"],
        gp(med["tmu"]), it, med["solve"], err_txt, oracle_s, oracle.num_threads()), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="0,1,2,3")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--reps", type=int, default=10)
    args = ap.parse_args()
    oracle.build()
    print("| config | precision | N | N_pair (R <= r_c) | slots evaluated per product | list build ms | field kernel ms "
          "(G pairs/s) | T.mu kernel ms (G pairs/s) | PCG iterations (1e-6) | solve ms | rel-L2 T.mu / E / mu, rel E_pol "
          "vs oracle | oracle + parity run s (cores) |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|")
    for c in [int(x) for x in args.configs.split(",") if x != ""]:
        s = make_config(c)
        for precision in (("fp64", "mixed") if c < 2 else ("mixed",)):
            run_one(s, str(c), precision, args.reps, full_oracle=c < 3)
    if args.sweep:
        for rc in (7.0, 9.0, 12.0):
            s = make_config(4, cutoff=rc)
            for precision in ("fp64", "mixed"):
                run_one(s, "4, r_c = %g A, beta = %.5f" % (rc, s.ewald_beta), precision, max(3, args.reps // 2),
                        full_oracle=True)


if __name__ == "__main__":
    main()
