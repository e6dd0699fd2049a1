#!/usr/bin/env python
"""bench.py -- headline benchmark of the real-space AMOEBA polarization hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 0|1|2|3] [--precision mixed|fp64] [--list-mode auto|tiles|cluster|atom]
    python bench.py --table [--table-configs 0,1,2,3] [--sweep] [--reps R]

One STEP = one pass of the whole hot path over one synthetic system:
neighbour-list build -> permanent field -> PCG solve to RMS 1e-6 -> polarization energy
(BASELINE.json configs[1] wording), by default on the 98,304-atom heterogeneous box
(configs[2], the system BASELINE.json's target is quoted on) in MIXED precision.

metric/unit: useful pair interactions per second.  One pair interaction = one unordered atom
pair {i,j} with R <= r_c evaluated once, for both atoms, in the field or in one T.mu product.
A step performs N_pair * (1 + n_matvec) of them (n_matvec = PCG iterations + 1 for the initial
residual); value = that / step time, summed over GPUs (replicas: SURVEY 8(e) "replicas only").

Prints ONE JSON line on rank 0 (see DESIGN.md section 7 for every key).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "useful pair interactions/s (field + T.mu matvecs of one list-build + field + PCG solve + energy step)"
UNIT = "pair interactions/s"
FLOPS_PER_PAIR_TMU = 89      # 32 FFMA*2 + 22 FMUL + 3 FADD per evaluated slot
FLOPS_PER_PAIR_FIELD = 160
# What the ATOM-list MIXED T.mu loop EXECUTES per evaluated slot (ordered pair), counted in the SASS of
# its rows (8 slots per row and lane) -- profiles/r02_sass_tmu_rows.txt, build named there:
#   FAR row : 44 FFMA2 + 24 FMUL2 + 8 FADD2 + 48 FFMA + 16 FMUL + 8 FADD, 16 MUFU
#   NEAR row: 68 FFMA2 + 44 FMUL2 + 8 FADD2 + 48 FFMA + 24 FMUL + 8 FADD, 32 MUFU
# FMA-pipe lane-cycles (a packed instruction holds the pipe 2 cycles) and FP32 flops per slot:
TMU_FAR_PIPE_CYCLES = (2 * (44 + 24 + 8) + 48 + 16 + 8) / 8
TMU_NEAR_PIPE_CYCLES = (2 * (68 + 44 + 8) + 48 + 24 + 8) / 8
TMU_FAR_FLOPS = (4 * 44 + 2 * 24 + 2 * 8 + 2 * 48 + 16 + 8) / 8
TMU_NEAR_FLOPS = (4 * 68 + 2 * 44 + 2 * 8 + 2 * 48 + 24 + 8) / 8
FP32_LANES_PER_SM = 128      # B200_PROFILING.md unit counts; FP64: half rate
WORKLOADS = {0: "cfg0_water648", 1: "cfg1_dhfr_size_23559", 2: "cfg2_hetero_98304", 3: "cfg3_stmv_size_1066629"}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[0, 1, 2, 3])
    ap.add_argument("--precision", default="mixed", choices=["mixed", "fp64", "fixed"])
    ap.add_argument("--list-mode", default="auto", choices=["auto", "tiles", "cluster", "atom"])
    ap.add_argument("--tol", type=float, default=1e-6)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-stored-t", action="store_true", help="skip the stored-matrix-elements leg (TKHP_SOLVER_STORED_T)")
    ap.add_argument("--peak-seconds", type=float, default=1.0)
    ap.add_argument("--no-other-configs", action="store_true",
                    help="skip the short legs on configs 0, 1, 3 (MIXED) and config 2 in FP64 / FIXED")
    ap.add_argument("--other-steps", type=int, default=10, help="timed steps of each short leg")
    ap.add_argument("--table", action="store_true",
                    help="instead of the JSON line: the markdown result table of BASELINE.md section 3 "
                         "(every config and precision, errors against the oracle; several minutes)")
    ap.add_argument("--table-configs", default="0,1,2,3")
    ap.add_argument("--sweep", action="store_true", help="--table: add config 4 (r_c = 7, 9, 12 A, both precisions)")
    ap.add_argument("--reps", type=int, default=10)
    return ap.parse_args()


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks/throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.lines: list[str] = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 9:
                continue
            try:
                sm.append(float(parts[1])); smax.append(float(parts[2])); power.append(float(parts[3]))
            except ValueError:
                continue
            for name, flag in zip(names, parts[5:9]):
                if flag.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(smax), "samples": len(sm),
                "power_w_max": max(power), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------- CPU oracle legs
def oracle_sample(sys_, n_rows: int, seed: int = 7):
    """Time the oracle as it stands on a bounded sample of rows: field + one T.mu on n_rows rows."""
    import oracle
    rng = np.random.default_rng(seed)
    rows = np.sort(rng.choice(sys_.n_atoms, size=min(n_rows, sys_.n_atoms), replace=False)).astype(np.int64)
    mu = rng.standard_normal((sys_.n_atoms, 3)) * 0.1
    ordered = oracle.count_pairs_rows(sys_, rows)          # not timed: the unit count
    t0 = time.perf_counter()
    oracle.perm_field_rows(sys_, rows)
    oracle.tmatvec_rows(sys_, mu, rows)
    dt = time.perf_counter() - t0
    # ordered evaluations / 2 = unordered-pair equivalents, times 2 operators
    return {"pair_interactions": float(ordered), "seconds": dt, "rows": int(rows.size),
            "cores": oracle.num_threads()}


def run_reference(args, rank: int, world: int):
    """--impl reference: the CPU oracle, as it stands, on this arm's config/metric (rank 0 only)."""
    if rank != 0:
        return
    from synth_inputs import make_config
    import oracle
    oracle.build()
    sys_ = make_config(args.config)
    n_rows = 2048 if sys_.n_atoms > 5000 else sys_.n_atoms
    for _ in range(min(args.warmup, 1)):
        oracle_sample(sys_, max(64, n_rows // 8))
    tot_pairs, tot_s = 0.0, 0.0
    cores = 1
    for k in range(args.steps):
        r = oracle_sample(sys_, n_rows, seed=100 + k)
        tot_pairs += r["pair_interactions"]; tot_s += r["seconds"]; cores = r["cores"]
    value = tot_pairs / tot_s
    sample = (f"each step: oracle perm_field + one tmatvec on {n_rows} seeded random rows of "
              f"{WORKLOADS[args.config]} (O(N) minimum-image loop per row, FP64)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config], "n_atoms": sys_.n_atoms, "cutoff": sys_.cutoff,
                   "ewald_beta": sys_.ewald_beta, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- result table
def _table_rows(s, perm, n_rand, n_blocks, seed=0):
    rng = np.random.default_rng(seed)
    rows = set(rng.choice(s.n_atoms, size=min(n_rand, s.n_atoms), replace=False).tolist())
    nb = perm.size // 32
    for b in rng.choice(nb, size=min(n_blocks, nb), replace=False):
        rows.update(int(a) for a in perm[32 * b:32 * b + 32] if a >= 0)
    rows.update(int(a) for a in perm[-32:] if a >= 0)
    return np.array(sorted(rows), dtype=np.int64)


def _table_one(s, label, precision, reps, full_oracle):
    """One row of the table: medians of `reps` steps (CUDA events inside the library), the live pair
    kernel durations, and the errors against the FP64 oracle (the cpu_baseline's oracle, as it stands)."""
    import torch
    import oracle
    import paper_2011_01207_b200 as pk
    rel = lambda a, b: float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(b))
    prec = pk.TKHP_FP64 if precision == "fp64" else pk.TKHP_MIXED
    stream = torch.cuda.Stream()
    torch.cuda.set_stream(stream)
    P = pk.Polarizer.for_system(s, precision=prec, list_mode=pk.TKHP_LIST_ATOM)
    dev = P.device
    f64 = torch.float64
    d_pos = torch.as_tensor(s.pos, dtype=f64, device=dev)
    d_alpha = torch.as_tensor(s.polarizability, dtype=f64, device=dev)
    d_group = torch.as_tensor(s.group_id, dtype=torch.int32, device=dev)
    probe = np.random.default_rng(1).standard_normal((s.n_atoms, 3)) * 0.1
    d_probe = torch.as_tensor(probe, dtype=f64, device=dev)
    t = dict(build=[], field=[], solve=[], energy=[], tmu=[], fld=[])
    it = 0
    for r in range(reps + 2):
        pk.tkhp_profile_reset(P.ctx, True)
        pk.tkhp_nblist_build(P.ctx, d_pos, d_alpha, d_group, stream)
        E = P.perm_field(s.charge, s.dipole, s.quad)
        mu, it, rms = P.polar_solve(E, tol=1e-6)
        float(P.polar_energy(mu, E).cpu())
        P.tmatvec(d_probe)                                  # one stand-alone product: the T.mu pair kernel's time
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
        err_txt = "%.1e / %.1e / %.1e, %.1e" % (rel(Tg, T_ref), rel(Eg.cpu().numpy(), E_ref),
                                                rel(mu_g.cpu().numpy(), mu_ref), abs(e_g - e_ref) / abs(e_ref))
    else:
        rows = _table_rows(s, perm, 2048, 8)
        err_txt = "%.1e / %.1e / -, - (%d sampled rows)" % (rel(Tg[rows], oracle.tmatvec_rows(s, probe, rows)),
                                                           rel(Eg.cpu().numpy()[rows], oracle.perm_field_rows(s, rows)), rows.size)
    oracle_s = time.perf_counter() - t0
    P.close()
    gp = lambda ms: n_pair / (ms * 1e-3) / 1e9
    print("| %s | %s | %d | %d | %d | %.3f | %.4f (%.0f) | %.4f (%.0f) | %d | %.3f | %s | %.0f (%d) |" % (
        label, precision, s.n_atoms, n_pair, n_slots, med["build"], med["fld"], gp(med["fld"]), med["tmu"],
        gp(med["tmu"]), it, med["solve"], err_txt, oracle_s, oracle.num_threads()), flush=True)


def run_table(args):
    """--table: BASELINE.md section 3's result table (SURVEY 8(d) protocol), markdown rows on stdout."""
    import oracle
    from synth_inputs import make_config
    oracle.build()
    print("| config | precision | N | N_pair (R <= r_c) | slots evaluated per product | list build ms | field kernel ms "
          "(G pairs/s) | stand-alone T.mu kernel ms (G pairs/s) | PCG iterations (1e-6) | solve ms | rel-L2 T.mu / E / mu, "
          "rel E_pol vs oracle | oracle + parity run s (cores) |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|")
    for c in [int(x) for x in args.table_configs.split(",") if x != ""]:
        s = make_config(c)
        for precision in (("fp64", "mixed") if c < 3 else ("mixed",)):
            _table_one(s, str(c), precision, args.reps, full_oracle=c < 3)
    if args.sweep:
        for rc in (9.0, 12.0):
            s = make_config(4, cutoff=rc)
            for precision in ("fp64", "mixed"):
                _table_one(s, "4, r_c = %g A, beta = %.5f" % (rc, s.ewald_beta), precision, max(3, args.reps // 2),
                           full_oracle=True)


# ----------------------------------------------------------------------------- our arm
def run_ours(args, rank: int, world: int, local_rank: int):
    import torch
    import paper_2011_01207_b200 as pk
    from paper_2011_01207_b200 import replicas
    from synth_inputs import make_config

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libtkhp has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist_mod.init_process_group("nccl", device_id=dev)
        dist = dist_mod

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sys_ = make_config(args.config)
    n = sys_.n_atoms
    precision = {"mixed": pk.TKHP_MIXED, "fp64": pk.TKHP_FP64, "fixed": pk.TKHP_FIXED}[args.precision]
    want_mode = {"auto": pk.TKHP_LIST_ATOM, "atom": pk.TKHP_LIST_ATOM, "cluster": pk.TKHP_LIST_CLUSTER,
                 "tiles": pk.TKHP_LIST_TILES}[args.list_mode]
    mode_name = {pk.TKHP_LIST_TILES: "tiles", pk.TKHP_LIST_CLUSTER: "cluster", pk.TKHP_LIST_ATOM: "atom"}
    P = pk.Polarizer.for_system(sys_, precision=precision, list_mode=want_mode, device=local_rank)
    f64 = torch.float64
    d_pos = torch.as_tensor(sys_.pos, dtype=f64, device=dev)
    d_alpha = torch.as_tensor(sys_.polarizability, dtype=f64, device=dev)
    d_group = torch.as_tensor(sys_.group_id, dtype=torch.int32, device=dev)
    d_q = torch.as_tensor(sys_.charge, dtype=f64, device=dev)
    d_dip = torch.as_tensor(sys_.dipole, dtype=f64, device=dev)
    d_quad = torch.as_tensor(sys_.quad, dtype=f64, device=dev)
    d_field = torch.empty((n, 3), dtype=f64, device=dev)
    d_mu = torch.empty((n, 3), dtype=f64, device=dev)
    d_energy = torch.empty((), dtype=f64, device=dev)
    torch.cuda.synchronize()
    # a stream of our own (the library replays its list build as a CUDA graph, which the legacy default
    # stream cannot capture); it is made torch's current stream, so the events below see it
    stream = torch.cuda.Stream(device=dev)
    torch.cuda.set_stream(stream)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def step():
        pk.tkhp_nblist_build(P.ctx, d_pos, d_alpha, d_group, stream)
        pk.tkhp_perm_field(P.ctx, d_q, d_dip, d_quad, d_field, stream)
        it, rms, ok = pk.tkhp_polar_solve(P.ctx, d_field, d_mu, args.tol, 100, False, stream)
        pk.tkhp_polar_energy(P.ctx, d_mu, d_field, d_energy, stream)
        return it, rms

    for _ in range(max(args.warmup, 3)):
        it, rms = step()
    torch.cuda.synchronize()
    n_pair, n_slots, mode_in_use = P.nblist_stats()
    energy = float(d_energy.cpu())

    # ---- timed region: K steps, device-resident inputs, L2 flushed between steps
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    pk.tkhp_profile_reset(P.ctx, True)
    prof_tot = dict(launches=0, n_tmatvec=0, tmatvec_ms=0.0, n_field=0, field_ms=0.0,
                    n_solve=0, solve_ms=0.0, solve_matvecs=0)
    iters, phases = [], []
    sampler.start()
    barrier()
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.fill_(k & 0xFF)
        ev[k][0].record(stream)
        it, rms = step()
        ev[k][1].record(stream)
        iters.append(it)
        pr = pk.tkhp_profile_read(P.ctx)
        pr.update(pk.tkhp_profile_read_solve(P.ctx))
        for key in prof_tot:
            prof_tot[key] += pr[key]
        phases.append(P.timings())
        pk.tkhp_profile_reset(P.ctx, True)
    barrier()
    wall_s = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = sum(step_ms)
    total_ms, wall_s = replicas.max_over_ranks([total_ms, wall_s], dist, dev)
    if not replicas.replicas_agree(statistics.mean(iters), energy, dist, dev):
        raise SystemExit("bench.py: replicas disagree on iteration count or energy")
    ms_per_step = total_ms / args.steps
    n_matvec = statistics.mean(iters) + 1
    pairs_per_step = n_pair * (1 + n_matvec)
    value = replicas.aggregate_throughput(pairs_per_step, world, ms_per_step)

    def stats(v):
        return {"mean": statistics.mean(v), "median": statistics.median(v), "min": min(v)}
    phase_names = ["build", "field", "tmatvec", "solve", "energy"]
    phase_ms = {nm: statistics.mean(ph[nm] for ph in phases) for nm in phase_names}
    phase_stats = {nm: stats([ph[nm] for ph in phases]) for nm in phase_names if nm != "tmatvec"}

    # ---- a stand-alone T.mu product (tkhp_tmatvec: pack + pair kernel + finish), 20 calls, L2 flushed
    d_probe = torch.as_tensor(np.random.default_rng(5).standard_normal((n, 3)) * 0.1, dtype=f64, device=dev)
    d_out = torch.empty((n, 3), dtype=f64, device=dev)
    for _ in range(3):
        pk.tkhp_tmatvec(P.ctx, d_probe, d_out, stream)
    pk.tkhp_profile_reset(P.ctx, True)
    mv_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(20)]
    for a_, b_ in mv_ev:
        flush.fill_(1)
        a_.record(stream)
        pk.tkhp_tmatvec(P.ctx, d_probe, d_out, stream)
        b_.record(stream)
    torch.cuda.synchronize()
    mv_call = [a_.elapsed_time(b_) for a_, b_ in mv_ev]
    mv_prof = pk.tkhp_profile_read(P.ctx)
    mv_kernel_ms = mv_prof["tmatvec_ms"] / max(mv_prof["n_tmatvec"], 1)
    phase_ms["tmatvec"] = statistics.median(mv_call)
    phase_stats["tmatvec"] = stats(mv_call)
    pk.tkhp_profile_reset(P.ctx, False)

    # ---- dominant kernel roofline, measured live with CUDA events on the library's stream
    props = torch.cuda.get_device_properties(dev)
    sm_count = props.multi_processor_count
    sm_ghz = 1.965
    try:
        sm_ghz = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())["sm_max_mhz"] / 1e3
    except Exception:
        if clocks.get("sm_max_mhz"):
            sm_ghz = clocks["sm_max_mhz"] / 1e3
    lanes_per_s = sm_count * FP32_LANES_PER_SM * sm_ghz * 1e9
    peak32 = 2 * lanes_per_s / 1e12
    peak = peak32 / 2 if args.precision == "fp64" else peak32
    fld_ms = prof_tot["field_ms"] / max(prof_tot["n_field"], 1)
    persistent = prof_tot["n_solve"] > 0
    if persistent:
        # the whole solve is ONE launch of k_pcg_persist: its T.mu products are the algorithmic work
        kern_ms = prof_tot["solve_ms"] / prof_tot["n_solve"]
        mv_per_launch = prof_tot["solve_matvecs"] / prof_tot["n_solve"]
        kernel_name = "%s (whole PCG solve: %.1f T.mu products + vector updates, one cooperative launch)" % (
            "k_pcg_persist" if mode_in_use == pk.TKHP_LIST_ATOM else "k_pcg_tiles", mv_per_launch)
        share = prof_tot["solve_ms"] / total_ms if world == 1 else None
        n_timed = prof_tot["n_solve"]
    else:
        kern_ms = prof_tot["tmatvec_ms"] / max(prof_tot["n_tmatvec"], 1)
        mv_per_launch = 1.0
        kernel_name = "T.mu pair kernel (%s list)" % mode_name[mode_in_use]
        share = prof_tot["tmatvec_ms"] / total_ms if world == 1 else None
        n_timed = prof_tot["n_tmatvec"]
    alg_flops = FLOPS_PER_PAIR_TMU * n_pair * mv_per_launch
    achieved = alg_flops / (kern_ms * 1e-3) / 1e12 if kern_ms > 0 else 0.0
    roofline = {
        "bound": "alu", "kernel": kernel_name,
        "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
        "traffic": None,
        "algorithmic_flops_per_launch": alg_flops, "matvecs_per_launch": mv_per_launch,
        "avg_launch_ms": kern_ms, "ms_per_matvec_in_kernel": kern_ms / mv_per_launch, "launches_timed": n_timed,
        "share_of_step": share,
        "executed_slots_per_matvec": n_slots,
        "useful_pairs_per_s_kernel": n_pair * mv_per_launch / (kern_ms * 1e-3) if kern_ms > 0 else 0.0,
        "field_kernel_avg_ms": fld_ms,
        "field_kernel_tflops": FLOPS_PER_PAIR_FIELD * n_pair / (fld_ms * 1e-3) / 1e12 if fld_ms > 0 else None,
        "peak_note": "%d SMs (queried) x %d FP32 lanes x 2 flop x %.3f GHz (MEASURED_PEAKS sm_max_mhz; DESIGN.md section 6)"
                     % (sm_count, FP32_LANES_PER_SM, sm_ghz),
        "standalone_tmatvec": {
            "kernel": "T.mu pair kernel (%s list), one launch per product" % mode_name[mode_in_use],
            "avg_kernel_ms": mv_kernel_ms, "launches_timed": mv_prof["n_tmatvec"],
            "achieved": FLOPS_PER_PAIR_TMU * n_pair / (mv_kernel_ms * 1e-3) / 1e12 if mv_kernel_ms > 0 else None,
            "frac": FLOPS_PER_PAIR_TMU * n_pair / (mv_kernel_ms * 1e-3) / 1e12 / peak if mv_kernel_ms > 0 else None,
            "call_ms": phase_stats["tmatvec"],
        },
    }
    if mode_in_use == pk.TKHP_LIST_ATOM and args.precision != "fp64":
        far, near, segs, far_on = P.nblist_atom_stats()
        if not far_on:
            near, far = far + near, 0
        pipe_cycles = TMU_FAR_PIPE_CYCLES * far + TMU_NEAR_PIPE_CYCLES * near
        flops_sass = TMU_FAR_FLOPS * far + TMU_NEAR_FLOPS * near
        roofline["executed_far_slots"] = far
        roofline["executed_near_slots"] = near
        roofline["executed_tflops_sass"] = flops_sass * mv_per_launch / (kern_ms * 1e-3) / 1e12
        roofline["fma_pipe_busy_frac"] = pipe_cycles * mv_per_launch / (kern_ms * 1e-3) / lanes_per_s
        roofline["sass_counts_from"] = "profiles/r02_sass_tmu_rows.txt"
    try:
        traffic_file = ROOT / "profiles" / "traffic.json"
        if traffic_file.exists():
            tj = json.loads(traffic_file.read_text())
            roofline["traffic"] = tj.get("k_pcg_persist" if persistent else mode_name[mode_in_use])
            roofline["traffic_note"] = tj.get("note")
    except Exception:
        pass
    # list build against the HBM roofline (~190 B/atom of prescribed traffic + the lists written)
    hbm_gbs = None
    try:
        hbm_gbs = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())["hbm_gbs"]
    except Exception:
        pass
    build_bytes = 190.0 * n + 2.0 * n_slots
    build_roofline = {"bound": "hbm", "algorithmic_bytes": build_bytes, "ms": phase_ms["build"],
                      "achieved_gbs": build_bytes / (phase_ms["build"] * 1e-3) / 1e9 if phase_ms["build"] > 0 else None,
                      "peak_gbs": hbm_gbs,
                      "frac": (build_bytes / (phase_ms["build"] * 1e-3) / 1e9 / hbm_gbs) if hbm_gbs and phase_ms["build"] > 0 else None,
                      "note": "190 B/atom (SURVEY 8(d)) + 2 B per list slot written"}

    # ---- the same product with STORED real-space matrix elements (TKHP_SOLVER_STORED_T; SURVEY 8(f) 1b,
    # PAPER.md L160-162): a second context on the same system, 20 products with the L2 flushed; the
    # stream (8 B per list slot + the 2 B list entry) is what bounds it, so it goes against the HBM roofline
    stored_t = None
    if (rank == 0 and world == 1 and not args.no_stored_t and mode_in_use == pk.TKHP_LIST_ATOM
            and args.precision != "fp64"):
        P2 = pk.Polarizer.for_system(sys_, precision=precision, list_mode=want_mode, device=local_rank,
                                     solver_flags=pk.TKHP_SOLVER_STORED_T)
        pk.tkhp_nblist_build(P2.ctx, d_pos, d_alpha, d_group, stream)
        for _ in range(3):
            pk.tkhp_tmatvec(P2.ctx, d_probe, d_out, stream)        # the first call also computes the elements
        pk.tkhp_profile_reset(P2.ctx, True)
        for _ in range(20):
            flush.fill_(1)
            pk.tkhp_tmatvec(P2.ctx, d_probe, d_out, stream)
        torch.cuda.synchronize()
        pr2 = pk.tkhp_profile_read(P2.ctx)
        st_ms = pr2["tmatvec_ms"] / max(pr2["n_tmatvec"], 1)
        pk.tkhp_profile_reset(P2.ctx, True)
        mu2 = torch.empty((n, 3), dtype=f64, device=dev)
        it2s, rms2s, _ = pk.tkhp_polar_solve(P2.ctx, d_field, mu2, args.tol, 100, False, stream)
        torch.cuda.synchronize()
        st_bytes = 10.0 * n_slots                                  # 8 B of factors + 2 B of list entry per slot
        stored_t = {"kernel": "k_atom_tmu_stored, one launch per product", "avg_kernel_ms": st_ms,
                    "launches_timed": pr2["n_tmatvec"], "bytes_per_product": st_bytes, "bound": "hbm",
                    "achieved_gbs": st_bytes / (st_ms * 1e-3) / 1e9 if st_ms > 0 else None,
                    "peak_gbs": hbm_gbs,
                    "frac": st_bytes / (st_ms * 1e-3) / 1e9 / hbm_gbs if hbm_gbs and st_ms > 0 else None,
                    "vs_recomputing_kernel_ms": mv_kernel_ms,
                    "solve_ms": P2.timings()["solve"], "solve_iterations": it2s,
                    "extra_workspace_bytes": P2.workspace_bytes - P.workspace_bytes}
        P2.close()

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).pin_memory()
        h_pos, h_alpha = pin(sys_.pos, f64), pin(sys_.polarizability, f64)
        h_group = pin(sys_.group_id, torch.int32)
        h_q, h_dip, h_quad = pin(sys_.charge, f64), pin(sys_.dipole, f64), pin(sys_.quad, f64)
        h_mu = torch.empty((n, 3), dtype=f64).pin_memory()
        h_e = torch.empty(1, dtype=f64).pin_memory()
        for _ in range(2):
            pk.tkhp_polarize_host(P.ctx, h_pos, h_alpha, h_group, h_q, h_dip, h_quad, args.tol, 100,
                                  h_mu, None, h_e, stream)
        barrier()
        e2e_ms, e2e_iters = [], []
        for k in range(args.steps):
            flush.fill_(k & 0xFF)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            it2, _, _ = pk.tkhp_polarize_host(P.ctx, h_pos, h_alpha, h_group, h_q, h_dip, h_quad,
                                              args.tol, 100, h_mu, None, h_e, stream)
            _ = float(h_e[0])
            e2e_ms.append((time.perf_counter() - t0) * 1e3)
            e2e_iters.append(it2)
        barrier()
        tot = sum(e2e_ms)
        (tot,) = replicas.max_over_ranks([tot], dist, dev)
        e2e_step = tot / args.steps
        e2e = {"value": replicas.aggregate_throughput(n_pair * (2 + statistics.mean(e2e_iters)), world, e2e_step),
               "unit": UNIT,
               "ms_per_step": e2e_step,
               "ms_per_step_stats": stats(e2e_ms),
               "h2d_bytes_per_step": n * (24 + 8 + 4 + 8 + 24 + 48),
               "d2h_bytes_per_step": n * 24 + 8}

    # ---- short legs on the other north_star systems and precisions (same step, same timing rules, L2 flushed;
    # BASELINE.json configs[0], [1], [3] in MIXED and the headline system in FP64 and FIXED), so that the
    # driver's one line carries them: ms per step, phases, iterations and the dominant kernel's fraction
    def short_leg(cfg, prec_name, steps):
        s2 = sys_ if cfg == args.config else make_config(cfg)
        prec2 = {"mixed": pk.TKHP_MIXED, "fp64": pk.TKHP_FP64, "fixed": pk.TKHP_FIXED}[prec_name]
        Q = pk.Polarizer.for_system(s2, precision=prec2, list_mode=pk.TKHP_LIST_ATOM, device=local_rank)
        n2 = s2.n_atoms
        t_ = lambda a, dt=f64: torch.as_tensor(a, dtype=dt, device=dev)
        a_pos, a_al, a_g = t_(s2.pos), t_(s2.polarizability), t_(s2.group_id, torch.int32)
        a_q, a_d, a_th = t_(s2.charge), t_(s2.dipole), t_(s2.quad)
        o_f = torch.empty((n2, 3), dtype=f64, device=dev)
        o_mu = torch.empty((n2, 3), dtype=f64, device=dev)
        o_e = torch.empty((), dtype=f64, device=dev)

        def one():
            pk.tkhp_nblist_build(Q.ctx, a_pos, a_al, a_g, stream)
            pk.tkhp_perm_field(Q.ctx, a_q, a_d, a_th, o_f, stream)
            it_, rms_, _ = pk.tkhp_polar_solve(Q.ctx, o_f, o_mu, args.tol, 100, False, stream)
            pk.tkhp_polar_energy(Q.ctx, o_mu, o_f, o_e, stream)
            return it_
        for _ in range(3):
            one()
        torch.cuda.synchronize()
        np2, ns2, mode2 = Q.nblist_stats()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        tot = dict(n_tmatvec=0, tmatvec_ms=0.0, n_solve=0, solve_ms=0.0, solve_matvecs=0, launches=0)
        its, phs = [], []
        pk.tkhp_profile_reset(Q.ctx, True)
        for k in range(steps):
            flush.fill_(k & 0xFF)
            evs[k][0].record(stream)
            its.append(one())
            evs[k][1].record(stream)
            pr_ = pk.tkhp_profile_read(Q.ctx)
            pr_.update(pk.tkhp_profile_read_solve(Q.ctx))
            for key in tot:
                tot[key] += pr_[key]
            phs.append(Q.timings())
            pk.tkhp_profile_reset(Q.ctx, True)
        torch.cuda.synchronize()
        ms = [a_.elapsed_time(b_) for a_, b_ in evs]
        if tot["n_solve"] > 0:
            k_ms = tot["solve_ms"] / tot["n_solve"]
            mv = tot["solve_matvecs"] / tot["n_solve"]
            k_name = "k_pcg_persist" if mode2 == pk.TKHP_LIST_ATOM else "k_pcg_tiles"
        else:
            k_ms = tot["tmatvec_ms"] / max(tot["n_tmatvec"], 1)
            mv = 1.0
            k_name = "T.mu pair kernel (%s list)" % mode_name[mode2]
        pk2 = peak32 / 2 if prec_name == "fp64" else peak32
        tf = FLOPS_PER_PAIR_TMU * np2 * mv / (k_ms * 1e-3) / 1e12 if k_ms > 0 else 0.0
        n_mv = statistics.mean(its) + 1
        out = {"workload": WORKLOADS[cfg], "precision": prec_name, "n_atoms": n2, "list_mode": mode_name[mode2],
               "steps": steps, "ms_per_step": statistics.mean(ms), "ms_per_step_stats": stats(ms),
               "phase_ms": {nm: statistics.mean(ph[nm] for ph in phs) for nm in ("build", "field", "solve", "energy")},
               "pcg_iterations": statistics.mean(its), "n_pair_within_cutoff": np2,
               "value": np2 * (1 + n_mv) / (statistics.mean(ms) * 1e-3), "unit": UNIT,
               "dominant_kernel": k_name, "dominant_kernel_avg_ms": k_ms, "matvecs_per_launch": mv,
               "dominant_kernel_tflops": tf, "dominant_kernel_frac": tf / pk2, "peak": pk2,
               "gpu_launches": tot["launches"], "energy_kcal_mol": float(o_e.cpu())}
        Q.close()
        return out

    other_configs = None
    if rank == 0 and world == 1 and not args.no_other_configs and args.config == 2 and args.precision == "mixed":
        other_configs = []
        for cfg, prec_name in ((0, "mixed"), (1, "mixed"), (3, "mixed"), (2, "fp64"), (2, "fixed")):
            try:
                other_configs.append(short_leg(cfg, prec_name, args.other_steps))
            except Exception as exc:        # a leg that fails is reported, it does not take the headline down
                other_configs.append({"workload": WORKLOADS[cfg], "precision": prec_name, "error": repr(exc)})
            torch.cuda.empty_cache()

    # ---- measured FMA peak and the CPU oracle beside it (rank 0, N = 1 only for the oracle)
    fma_peak = pk.tkhp_fma_peak(local_rank, precision, args.peak_seconds) if rank == 0 else None
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        rows = min(n, 131072)        # config 2: every row once, about 7 s on 16 cores
        r = oracle_sample(sys_, rows)
        cpu = {"value": r["pair_interactions"] / r["seconds"], "unit": UNIT, "cores": r["cores"],
               "kind": "oracle", "seconds": r["seconds"],
               "sample": f"oracle perm_field + one tmatvec on {r['rows']} seeded random rows of {WORKLOADS[args.config]}"}
    P.close()
    if dist is not None:
        dist.destroy_process_group()
    if rank != 0:
        return
    if roofline is not None and fma_peak:
        roofline["peak_measured_fma_chain"] = fma_peak
        roofline["frac_of_measured_fma"] = achieved / fma_peak
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": {"mixed": "f32 pair math, f64 accumulation", "fp64": "f64",
                  "fixed": "f32 pair math, int64 fixed-point accumulation"}[args.precision],
        "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config], "n_atoms": n, "box": sys_.box,
                   "cutoff": sys_.cutoff, "skin": sys_.skin, "ewald_beta": sys_.ewald_beta,
                   "tol": args.tol, "precision": args.precision,
                   "list_mode": mode_name[mode_in_use],
                   "parallelism": "replicas x%d" % world, "l2": "flushed between timed steps (256 MiB fill)"},
        "n_pair_within_cutoff": n_pair, "pcg_iterations": statistics.mean(iters),
        "pair_interactions_per_step": pairs_per_step, "energy_kcal_mol": energy, "final_rms": rms,
        "phase_ms": phase_ms, "phase_ms_stats": phase_stats, "step_ms_stats": stats(step_ms),
        "build_roofline": build_roofline,
        "launch_bound": n < 5000,
        "wall_ms_per_step_incl_flush": 1e3 * wall_s / args.steps,
        "roofline": roofline, "stored_t": stored_t, "cpu_baseline": cpu, "e2e": e2e,
        "other_configs": other_configs,
        "gpu_launches": prof_tot["launches"], "clocks": clocks,
    }
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world == 1 and args.gpus > 1 and args.impl == "ours":
        # plain `python bench.py --gpus N`: re-launch under torchrun, one rank per GPU
        from paper_2011_01207_b200 import replicas
        cmd = replicas.torchrun_command(sys.executable, str(Path(__file__).resolve()), args.gpus, sys.argv[1:])
        raise SystemExit(subprocess.call(cmd))
    if args.table:
        if rank == 0:
            run_table(args)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
