#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path on synthetic inputs.

One "step" = cell lists + cached near field + cached spread/gather lists, the induced-charge Krylov solve (eq. 13), the
final potential+field evaluation, forces / torques / energies -- i.e. set_positions + solve + forces through the C ABI.
metric = Ewald operator applications per second over whole steps; the two flavours differ 3-12x in work and are also
reported separately: M1 = bead-only solver matvec (psi at the conductor beads), M2 = full evaluation (all particles; psi
for the right-hand side, psi + E for the forces).  ms_per_step = whole step; solve.solve_ms_per_step = the Krylov solve
alone (BASELINE.json's second headline number).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

N > 1 (torchrun): the path does not shard (replicas only) -- every rank runs an
independent replica with its own seed; value is the sum over ranks, time the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC, UNIT = "ewald_matvecs_per_s", "matvec/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config index 1..5 (default 5: 500k beads + 1M ions)")
    ap.add_argument("--tol", type=float, default=1e-10, help="Ewald tolerance (xi, r_c, P follow eqs. 23, 28, 32)")
    ap.add_argument("--P", type=int, default=0)
    ap.add_argument("--tol-solver", type=float, default=1e-12)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-samples", type=int, nargs=2, default=None, help="two target counts for the oracle timing")
    ap.add_argument("--P-matvec", type=int, default=0, help="narrower window for the solver matvec (pce_params.P_matvec; default: P)")
    ap.add_argument("--deterministic", action="store_true", help="PCE_FLAG_DETERMINISTIC: bit-reproducible gather (no fp64 atomics)")
    ap.add_argument("--fig3d", action="store_true",
                    help="the paper's timing workload (PAPER.md:325, Fig. 3d): induced-charge solve of FCC arrays vs total bead count; "
                         "prints its own JSON line and exits")
    ap.add_argument("--no-configs", action="store_true", help="skip the short runs of BASELINE.json configs 1-4 reported in 'configs'")
    ap.add_argument("--bd", type=int, default=0, metavar="STEPS",
                    help="also run STEPS Brownian-dynamics steps on the device (solve + forces + pce_bd_step; config 3: 100, dt = 1e-4 a^2)")
    return ap.parse_args()


def make_workload(idx, rank=0):
    import workloads as wl
    seed = wl.configs.BASE_SEED + idx + 1000 * rank
    if idx == 1:
        return wl.config1()
    if idx == 2:
        return wl.config2(d=3.0, seed=seed)
    if idx == 3:
        return wl.config3(seed=seed)
    if idx == 4:
        return wl.config4(seed=seed)
    return wl.config5(seed=seed)


def ewald_params(L, Ng, a, tol, P=0):
    """(xi, r_c, P) from a tolerance by eqs. 28, 23 (+2a for shells, reading A14) and 32 -- the arithmetic the
    header states for pce_suggest_params, restated here so that the reference arm can describe its configuration without loading
    the product library (tests/test_abi.py holds the two to each other)."""
    import math
    L = np.broadcast_to(np.asarray(L, dtype=np.float64), (3,))
    Ng = np.broadcast_to(np.asarray(Ng), (3,))
    s = math.sqrt(-math.log(tol))
    kc = min(math.pi * (int(n) - 1) / float(l) for n, l in zip(Ng, L))
    xi = kc / (2.0 * s)
    rc = s / xi + 2.0 * a
    if P <= 0:
        P = 2 * math.ceil(((2.0 / math.pi) * (-math.log(tol)) + 4.0) / 2.0)
    P = min(max(P, 4), 32)
    for n in Ng:
        if P > int(n):
            P = int(n) & ~1
    return xi, rc, int(P)


def config_dict(w, args):
    """The `config` object of the JSON line: the workload and the Ewald parameters that follow from it (pure host arithmetic),
    identical in both arms so that the driver can pair them.  No import of the product package: the reference arm calls this."""
    xi, rc, P = ewald_params(w.L, w.Ng, w.a, args.tol, args.P)
    grid_bytes = 8 * int(np.prod(w.Ng))
    return {"workload": w.name, "N": w.N, "N_bead": w.N_bead, "N_body": w.N_body, "grid": [int(g) for g in w.Ng],
            "P": P, "P_matvec": int(args.P_matvec or P), "xi": xi, "rc": rc, "ewald_tol": args.tol, "solver_tol": args.tol_solver,
            "l2": "flushed between timed steps" if grid_bytes < 256 << 20 else "inputs larger than L2 (grids %.2f GB)" % (grid_bytes * 3 / 1e9),
            "multi_gpu": "replicas only"}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


# ---------------------------------------------------------------- clocks
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, dev):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(dev), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "200"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(",") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, reasons = [], set()
        for r in rows:
            try:
                sm.append(float(r[0])); out["sm_max_mhz"] = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if "Active" in v and "Not" not in v:
                    reasons.add(name)
        if sm:
            out["sm_mhz"] = float(np.median(sm))
        out["reasons"] = sorted(reasons)
        out["samples"] = len(sm)
        return out


# ---------------------------------------------------------------- oracle timing (cpu_baseline / --impl reference)
def oracle_matvec_seconds(w, samples, flavour="bead", seed=0):
    """Time the oracle (as it stands) on a bounded sample: potentials (flavour 'bead': bead sources and
    targets, potential only; 'full': all particles, potential + field) at S1 and S2 random targets from
    ALL sources; t(S) = A + B S is extrapolated to every target.  Small configs are timed in full."""
    import oracle as orc
    rng = np.random.default_rng(seed)
    if flavour == "bead":
        x, field = w.x[:w.N_bead], False
    else:
        x, field = w.x, True
    n = x.shape[0]
    q = rng.normal(size=n)
    if n <= 3000:
        t0 = time.perf_counter()
        orc.ewald_eval(x, q, w.L, w.a, w.eps_f, field=field)
        dt = time.perf_counter() - t0
        return dt, f"full {flavour} matvec, {n} targets", dt
    ts = []
    for S in samples:
        tg = rng.choice(n, size=S, replace=False)
        t0 = time.perf_counter()
        orc.ewald_eval(x, q, w.L, w.a, w.eps_f, targets=tg, field=field)
        ts.append(time.perf_counter() - t0)
    B = (ts[1] - ts[0]) / (samples[1] - samples[0])
    A = ts[0] - B * samples[0]
    if B <= 0:  # noise: fall back to proportional scaling of the larger sample
        A, B = 0.0, ts[1] / samples[1]
    full = max(A, 0.0) + B * n
    return full, f"{flavour} matvec at {samples[0]} and {samples[1]} of {n} targets from all {n} sources, t = A + B*S extrapolated to {n}", sum(ts)


def default_samples(w):
    # at least 4x the core count: the oracle parallelises over targets
    if w.N > 500000:
        return (64, 192)
    if w.N > 50000:
        return (128, 384)
    return (256, 768)


def run_reference(args, rank, world):
    """The oracle timed on the host cores (the reference arm of this tier).  Rank 0 only."""
    if rank != 0:
        return
    import oracle as orc
    orc.build()
    w = make_workload(args.config)
    samples = tuple(args.cpu_samples) if args.cpu_samples else default_samples(w)
    secs, spent_total, budget_s = [], 0.0, 150.0  # the whole run stays within a few minutes on any host
    n_total = args.warmup + args.steps
    for i in range(n_total):
        full, desc, spent = oracle_matvec_seconds(w, samples, "bead" if w.N_bead else "full", seed=i)
        spent_total += spent
        # samples that cost real time are all kept (a warm-up changes nothing for a pure CPU loop of tens of seconds)
        if i >= args.warmup or spent > 5.0:
            secs.append(full)
        remaining = n_total - i - 1
        if secs and remaining and spent_total + spent > budget_s:
            break
    t = float(np.mean(secs))
    val = 1.0 / t
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": config_dict(w, args),
        "counts": "one direct-sum M1 application (bead sources and targets, potential only) per step",
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
                         "sample": "direct-sum oracle, " + desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


# ---------------------------------------------------------------- replicas (multi-GPU: no sharding)
def reduce_over_ranks(dist, ms, count, device):
    """Whole-job figures of N independent replicas: (max over ranks of the timed ms, sum over ranks of the count).
    `dist` is an initialised torch.distributed module (nccl on GPUs; gloo in the CPU tests) or None for one rank."""
    if dist is None:
        return float(ms), float(count)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([count], dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), float(c.item())


def m1_algorithmic_bytes(w, nnz_near):
    """Algorithmic bytes of one bead-only matvec: spread, two transforms, scale, gather, cached near field."""
    Ng3, Nk = int(np.prod(w.Ng)), int((w.Ng[0] // 2 + 1) * w.Ng[1] * w.Ng[2])
    return (32 * w.N_bead + 8 * Ng3) + 2 * (8 * Ng3 + 16 * Nk) + 32 * Nk + (8 * Ng3 + 40 * w.N_bead) + 12 * nnz_near + 20 * w.N_bead


def small_config_row(pce, torch, idx, args, hbm_peak, steps=10, warmup=3):
    """One of BASELINE.json's smaller configurations through the same whole step (set_positions + solve + forces), on a stream
    of its own so that the solver's CUDA graph replays; L2 flushed between timed steps (their meshes fit in it)."""
    w = make_workload(idx)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        ctx = pce.context_for(w, tol=args.tol, P=args.P, tol_solver=args.tol_solver, stream=st)
        x, y, z, Q, qi = pce.upload(w)
        ctx.set_system(w.body_offset, x, y, z)
        info = ctx.info()
        flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
        ms, its, replays, conv, resid = [], [], 0, True, 0.0
        for i in range(warmup + steps):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            ctx.set_positions(x, y, z)
            q, Phi, si = ctx.solve(Q, qi, w.E0, allow_noconv=True)
            ctx.forces(q, w.E0)
            b.record()
            torch.cuda.synchronize()
            if i >= warmup:
                ms.append(a.elapsed_time(b)); its.append(si["iters"]); replays += si["graph_replays"]
                conv = conv and bool(si["converged"]); resid = max(resid, si["rel_resid"])
        row = {"config": idx, "workload": w.name, "N": w.N, "N_bead": w.N_bead, "grid": [int(g) for g in w.Ng], "fft_mode": info["fft_mode"],
               "ms_per_step": float(np.mean(ms)), "cg_iters": float(np.mean(its)), "converged": conv, "rel_resid": resid,
               "graph_replays_per_step": replays / steps, "steps": steps}
        if w.N_bead:
            qb = torch.randn(w.N_bead, dtype=torch.float64, device="cuda")
            ctx.matvec(qb)
            reps = 50
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a.record()
            for _ in range(reps):
                ctx.matvec(qb)
            b.record()
            torch.cuda.synchronize()
            m1 = a.elapsed_time(b) / reps
            nbytes = m1_algorithmic_bytes(w, info["nnz_near"])
            row.update({"m1_ms": m1, "m1_per_s": 1e3 / m1, "m1_frac_of_hbm_ceiling": (nbytes / (m1 * 1e-3)) / (hbm_peak * 1e9),
                        "m1_note": "back-to-back applications, mesh resident in L2 at these sizes"})
            row["value"] = float(np.sum(its)) / (float(np.sum(ms)) * 1e-3)  # M1 applications per second of whole steps, as the headline
        ctx.close()
    torch.cuda.synchronize()
    return row


# ---------------------------------------------------------------- our arm
def run_ours(args, rank, world, local_rank):
    import torch
    import paper_2401_04865_b200 as pce

    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local_rank))
    if rank == 0:
        pce.build()
    if dist:
        dist.barrier()
    # a stream of our own: the legacy default stream cannot be captured, and the solver replays its iteration as a CUDA graph
    # (solve.graph_replays says whether it did); everything below -- torch copies, events, the library -- is enqueued on it
    stream = torch.cuda.Stream()
    torch.cuda.set_stream(stream)
    w = make_workload(args.config, rank)
    ctx = pce.context_for(w, tol=args.tol, P=args.P, tol_solver=args.tol_solver, deterministic=args.deterministic, P_matvec=args.P_matvec,
                          stream=stream)
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    info = ctx.info()
    hbm_peak, peak_src, _ = peaks()
    grid_bytes = 8 * int(np.prod(w.Ng))
    l2_flush = None
    if grid_bytes < 256 << 20:  # working set may sit in the 126 MB L2: flush between timed steps
        l2_flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")

    def step(timed):
        ctx.set_positions(x, y, z)
        t_cells = ctx.timings() if timed else None
        q, Phi, sinfo = ctx.solve(Q, qi, w.E0, allow_noconv=True)
        t_solve = ctx.timings() if timed else None
        out = ctx.forces(q, w.E0)
        t_force = ctx.timings() if timed else None
        return q, out, sinfo, (t_cells, t_solve, t_force)

    sampler = ClockSampler(local_rank) if rank == 0 else None  # started before the warm-up: its start-up cost stays out of the timed steps
    for _ in range(args.warmup):
        step(False)
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    # ---- timed region: K whole steps, per-pass event timing OFF (no instrumentation inside the headline number)
    l0 = ctx.launch_count()
    ms_steps, iters, n_apply, n_m1, n_graph, all_converged = [], [], 0, 0, 0, True
    for _ in range(args.steps):
        if l2_flush is not None:
            l2_flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        q, out, sinfo, _ = step(False)
        e1.record()
        torch.cuda.synchronize()
        ms_steps.append(e0.elapsed_time(e1))
        iters.append(sinfo["iters"])
        n_apply += sinfo["matvecs"] + 1  # solver matvecs + right-hand-side evaluation, + the force evaluation
        n_m1 += sinfo["iters"]           # the bead-only solver matvecs alone: what the reference arm counts
        n_graph += sinfo["graph_replays"]
        all_converged = all_converged and bool(sinfo["converged"])
    launches = ctx.launch_count() - l0
    clocks = sampler.stop() if sampler else None
    # ---- the same K steps again with the library's per-pass CUDA events on: per-kernel durations for the rooflines
    ctx.set_timing(True)
    acc = {}
    ms_solve = []
    for _ in range(args.steps):
        if l2_flush is not None:
            l2_flush.fill_(1)
        torch.cuda.synchronize()
        q, out, sinfo, tms = step(True)
        torch.cuda.synchronize()
        for t in tms:
            for k, v in t.items():
                acc[k] = acc.get(k, 0) + v
        ms_solve.append(tms[1]["total"])
    ctx.set_timing(False)
    total_ms = float(sum(ms_steps))
    _, n_m1_all = reduce_over_ranks(dist, total_ms, n_m1, "cuda")
    total_ms, n_apply_all = reduce_over_ranks(dist, total_ms, n_apply, "cuda")
    # headline: M1 applications (bead-only solver matvecs, the unit the reference arm times) per second of WHOLE steps -- the two
    # full evaluations, the list rebuilds and the force pass of every step are in the denominator and count for nothing above it
    value = n_m1_all / (total_ms * 1e-3)
    value_all = n_apply_all / (total_ms * 1e-3)

    # ---- the two operator flavours on their own (CUDA events around back-to-back applications, this stream)
    def time_op(fn, reps):
        fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps
    flavours = {}
    reps = 10 if w.N > 100000 else 50
    if w.N_bead:
        qb = torch.randn(w.N_bead, dtype=torch.float64, device="cuda")
        ms1 = time_op(lambda: ctx.matvec(qb), reps)
        flavours["m1_bead_matvec"] = {"ms": ms1, "per_s": 1e3 / ms1, "what": "psi = M_bb q at the conductor beads (cached near field + spread/FFT/scale/IFFT/gather)"}
    qa = torch.randn(w.N, dtype=torch.float64, device="cuda")
    ms2 = time_op(lambda: ctx.evaluate(qa, field=True), max(reps // 5, 2))
    flavours["m2_full_evaluation"] = {"ms": ms2, "per_s": 1e3 / ms2, "what": "psi and E at all N particles from all N charges"}
    flavours["per_step"] = {"m1": float(np.mean(iters)), "m2": 2.0}

    # ---- optional: Brownian dynamics on the device: solve (cold / warm start) + forces + pce_bd_step per step
    bd = None
    if args.bd > 0 and w.N_ion > 0:
        dt_bd = 1e-4 * w.a ** 2
        bd = {"steps": args.bd, "dt": dt_bd, "what": "pce_solve + pce_forces + pce_bd_step per step, positions never leave the device"}
        for mode in ("cold", "warm"):
            ctx.set_positions(x, y, z)
            qprev, its = None, []
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for s_ in range(args.bd):
                qq, _, si = ctx.solve(Q, qi, w.E0, q0=qprev if mode == "warm" else None, allow_noconv=True)
                oo = ctx.forces(qq, w.E0)
                ctx.bd_step(oo["f"], dt_bd, 1.0, 1.0, seed=20240104 + args.config, step=s_)
                qprev = qq
                its.append(si["iters"])
            b.record()
            torch.cuda.synchronize()
            bd[mode] = {"ms_per_step": a.elapsed_time(b) / args.bd, "cg_iters_mean": float(np.mean(its))}
        ctx.set_positions(x, y, z)

    # ---- end to end through the host-buffer call (H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        def pin(a):
            return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).pin_memory()
        hx, hy, hz = pin(w.x[:, 0]), pin(w.x[:, 1]), pin(w.x[:, 2])
        hQ, hqi = pin(w.Q_body), pin(w.q_ion)
        nb = w.N_body
        outb = {"q": pin(np.zeros(w.N)), "Phi": pin(np.zeros(max(nb, 1))), "fx": pin(np.zeros(w.N)), "fy": pin(np.zeros(w.N)),
                "fz": pin(np.zeros(w.N)), "F": pin(np.zeros(max(3 * nb, 1))), "T": pin(np.zeros(max(3 * nb, 1))),
                "S": pin(np.zeros(max(3 * nb, 1))), "U": pin(np.zeros(3))}
        ctx.step_host(hx, hy, hz, hQ, hqi, w.E0, outb)  # warm
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        t0 = time.perf_counter()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        n_e2e = 0
        for _ in range(args.steps):
            si = ctx.step_host(hx, hy, hz, hQ, hqi, w.E0, outb)
            n_e2e += si["iters"]
        ev1.record()
        torch.cuda.synchronize()
        ms = max(ev0.elapsed_time(ev1), 1e3 * (time.perf_counter() - t0))  # the call is synchronous: host clock bounds it
        ms, n_e2e = reduce_over_ranks(dist, ms, n_e2e, "cuda")
        e2e = {"value": n_e2e / (ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 8 * (3 * w.N + nb + w.N_ion),
               "d2h_bytes_per_step": 8 * (w.N + nb + 3 * w.N + 9 * nb + 3), "ms_per_step": ms / args.steps}
    # ---- the other configurations of BASELINE.json, briefly (default run only: one GPU, config 5 as the headline)
    cfg_rows = None
    if world == 1 and args.config == 5 and not args.no_configs:
        cfg_rows = [small_config_row(pce, torch, i, args, hbm_peak) for i in (1, 2, 3, 4)]
    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    # ---- per-pass rooflines (algorithmic bytes of SURVEY.md 8(d), stated in DESIGN.md)
    Ng3, Nk = int(np.prod(w.Ng)), int((w.Ng[0] // 2 + 1) * w.Ng[1] * w.Ng[2])
    nm1, nfull = max(acc["n_matvec_bead"], 1), max(acc["n_eval_full"], 1)
    npairs = max(acc["n_fft_pairs"], 1)

    dfma_tf, dmma_tf = pce.measure_fp64_peaks()  # live, on this device (csrc/peaks.cu)
    P3 = float(ctx.params.P) ** 3
    P3b = float(info["P_matvec"]) ** 3   # the solver matvec spreads / gathers with its own, narrower window (pce.h: P_matvec)

    def rf(ms_total, launches_, bytes_per_launch, fma_per_launch=None):
        """HBM roofline of a pass; passes bound by fp64 arithmetic (fma_per_launch given: useful window updates, 2 flop each)
        report "bound": "alu" against the measured fp64 mma peak and keep the HBM figures beside it."""
        if ms_total <= 0:
            return None
        sec = ms_total / launches_ * 1e-3
        gbs = bytes_per_launch / sec / 1e9
        d = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
             "ms_per_launch": ms_total / launches_, "algorithmic_bytes": bytes_per_launch, "launches": launches_}
        if fma_per_launch:
            tf = 2.0 * fma_per_launch / sec / 1e12
            d.update({"bound": "alu", "achieved": tf, "peak": dmma_tf, "unit": "TFLOP/s", "frac": tf / dmma_tf,
                      "hbm_achieved_gbs": gbs, "hbm_frac": gbs / hbm_peak, "algorithmic_fma": fma_per_launch})
        return d
    # the (x, y) transforms (3-D transforms in mode 0) are cuFFT's unless the library runs its own passes (fftxy.cu)
    fft_keys = ("fft_xy_forward(own)", "fft_xy_inverse(own)") if info["fft_mode"] == 2 else ("fft_d2z(cuFFT)", "ifft_z2d(cuFFT)")
    fft_text = {0: "cuFFT 3-D D2Z/Z2D + separate scale pass",
                1: "cuFFT 2-D D2Z/Z2D per mesh plane; the 'scale' pass is the fused z FFT + Green's function + inverse z FFT kernel",
                2: "own (x, y) passes per mesh plane (fftxy.cu: one HBM trip per plane and direction); the 'scale' pass is the fused "
                   "z FFT + Green's function + inverse z FFT kernel; no library call on the path"}[info["fft_mode"]]
    # HBM ceiling of the bead-only matvec: the algorithmic bytes of all its passes at the measured copy rate
    m1_bytes = m1_algorithmic_bytes(w, info["nnz_near"])
    if "m1_bead_matvec" in flavours:
        flavours["m1_bead_matvec"].update({"algorithmic_bytes": m1_bytes, "hbm_ceiling_per_s": hbm_peak * 1e9 / m1_bytes,
                                           "frac_of_hbm_ceiling": flavours["m1_bead_matvec"]["per_s"] * m1_bytes / (hbm_peak * 1e9)})
    passes = {
        "spread_bead": rf(acc["bead_spread"], nm1, 32 * w.N_bead + 8 * Ng3, w.N_bead * P3b),
        "gather_bead": rf(acc["bead_gather"], nm1, 8 * Ng3 + 40 * w.N_bead, w.N_bead * P3b),
        "real_bead_csr": rf(acc["bead_real"], nm1, 12 * info["nnz_near"] + 20 * w.N_bead),
        "scale": rf(acc["scale"], npairs, 32 * Nk),
        fft_keys[0]: rf(acc["fft"], npairs, 8 * Ng3 + 16 * Nk),
        fft_keys[1]: rf(acc["ifft"], npairs, 8 * Ng3 + 16 * Nk),
        "spread_full": rf(acc["spread"] - acc["bead_spread"], nfull, 32 * w.N + 8 * Ng3, w.N * P3),
        # per step: one potential-only gather at the beads (right-hand side) and one potential + field gather at all N
        "gather_full": rf(acc["gather"] - acc["bead_gather"], nfull, 8 * Ng3 + (40 * w.N_bead + 64 * w.N) / 2,
                          (w.N_bead + 4 * w.N) / 2 * P3),
    }
    own = {k: v for k, v in passes.items() if v and "cuFFT" not in k}
    dom = max(own, key=lambda k: own[k]["ms_per_launch"] * own[k]["launches"])
    roof = dict(own[dom])
    roof["kernel"] = dom
    roof["peak_source"] = ("pce_measure_fp64_peaks (csrc/peaks.cu: fp64 mma.sync chains on this device, this run)" if roof["bound"] == "alu"
                           else peak_src)
    roof["traffic"] = None  # dram bytes per launch from the committed ncu --set full capture (config 5 only)
    tpath = os.path.join(ROOT, "profiles", "r2_traffic.json")
    if args.config == 5 and os.path.exists(tpath):
        roof["traffic"] = json.load(open(tpath)).get(dom)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "solve_converged": bool(all_converged), "solve_rel_resid": sinfo["rel_resid"], "solve_graph_replays_per_step": n_graph / args.steps,
        "value_all_flavours": value_all,
        "config": config_dict(w, args),
        "run_info": {"cells": info["ncell"], "nnz_near": info["nnz_near"], "deterministic_gather": bool(args.deterministic),
                     "fft": fft_text},
        "counts": "value = M1 bead-only solver matvecs / whole-step time (same unit as the reference arm; e2e likewise); "
                  "value_all_flavours adds the 2 full evaluations of every step to the numerator; the flavours are timed alone in 'flavours'",
        "flavours": flavours,
        "solve": {"cg_iters": iters, "solve_ms_per_step": float(np.mean(ms_solve)), "matvecs_bead": acc["n_matvec_bead"],
                  "evals_full": acc["n_eval_full"], "rel_resid": sinfo["rel_resid"], "converged": sinfo["converged"]},
        "passes_ms_per_step": {k: acc[k] / args.steps for k in ("cells", "real", "spread", "fft", "scale", "ifft", "gather", "krylov", "other", "total")},
        "passes_timed": "per-pass CUDA events of the library, in K instrumented repeats of the timed steps (the timed steps themselves carry no instrumentation)",
        "roofline": roof, "roofline_passes": passes,
        "fp64_peaks_tflops": {"dfma": dfma_tf, "mma_f64": dmma_tf, "how": "pce_measure_fp64_peaks: register-resident chains, this device, this run"}, "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e,
    }
    if bd:
        line["bd"] = bd
    if cfg_rows:
        line["configs"] = cfg_rows
    if not args.no_cpu_baseline:
        import oracle as orc
        orc.build()
        samples = tuple(args.cpu_samples) if args.cpu_samples else default_samples(w)
        t1, d1, _ = oracle_matvec_seconds(w, samples, "bead" if w.N_bead else "full")
        line["cpu_baseline"] = {"value": 1.0 / t1, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
                                "sample": "direct-sum oracle (one M1 application: bead sources and targets, potential only), " + d1,
                                "seconds_per_matvec": t1}
    print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


def run_fig3d(args):
    """Time per induced-charge solve of FCC arrays of ideally polarizable spheres in a uniform field, no ions (the shape of the
    paper's Fig. 3d: N_b = 8 ... 512 bodies x N = 42 ... 2562 beads, spectral-Ewald tolerance 1e-3, GTX 1080;
    here 4 m^3 bodies, reading B9), at the paper's tolerance and at this build's parity settings."""
    import torch
    import paper_2401_04865_b200 as pce
    import workloads as wl
    pce.build()
    rows = []
    for m, subdiv in ((1, 3), (2, 3), (3, 3), (4, 3), (5, 3), (2, 4), (3, 4), (4, 4)):
        w = wl.fcc_array(m, subdiv)
        for tol, tol_solver in ((1e-3, 1e-3), (1e-10, 1e-12)):
            ctx = pce.context_for(w, tol=tol, tol_solver=tol_solver)
            x, y, z, Q, qi = pce.upload(w)
            ctx.set_system(w.body_offset, x, y, z)
            ts, its = [], []
            for rep in range(4):
                torch.cuda.synchronize()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                ctx.set_positions(x, y, z)
                q, Phi, si = ctx.solve(Q, qi, w.E0, allow_noconv=True)
                b.record()
                torch.cuda.synchronize()
                if rep:
                    ts.append(a.elapsed_time(b)); its.append(si["iters"])
            rows.append({"bodies": w.N_body, "beads_per_body": w.N_bead // w.N_body, "N_T": w.N_bead, "grid": int(w.Ng[0]),
                         "P": int(ctx.params.P), "ewald_tol": tol, "solver_tol": tol_solver, "iters": int(np.median(its)),
                         "ms_per_solve": float(np.median(ts)), "converged": bool(si["converged"]), "fft_mode": ctx.info()["fft_mode"]})
            ctx.close()
    print(json.dumps({"fig3d": rows, "what": "ms per time step = cell lists + caches + induced-charge solve (cold start), FCC arrays, phi = 0.2, E0 = (0,0,1)"}))


def main():
    args = parse()
    if args.fig3d:
        return run_fig3d(args)
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    local_rank = int(os.environ.get("LOCAL_RANK", 0))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
