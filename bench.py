"""bench.py -- H-HIGNN mobility apply U = M(X) F on B200: particles/s of one whole hot-path step.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3|c4|c2|c1] [--impl reference]

A "step" is one pass of the whole hot path (hh_step): Morton keys, radix sort, cluster
tree, boxes, Alg. 1 block lists, Alg. 2 (ACA) factors streamed through the arena, near-field, far-field,
three-body, self term, Euler update, on one batch of synthetic input.  Default
workload at N=1 is BASELINE.json configs[2] ("c3": 1,048,576 particles, eta=1, zeta=1e-4), the 1M-particle
point the metric is quoted on; --workload c4 is the 10M point.  One JSON line is printed by rank 0.

The path does not shard (north_star: one GPU, no collectives; replicas only): with
--gpus N every rank runs an independent replica of the same step on its own seeded cloud and `value` is
the units all ranks processed / max-over-ranks time ("scaling": "weak").

--impl reference times the CPU oracle (oracle/, fp64, as it stands) on a bounded sample of the same
workload on the host cores; it is a deliberately slow program, a reported baseline and not the target.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "H-matvec particles/s (whole step: tree + blocks + ACA + near + far + three-body)"
UNIT = "particles/s"
FAR_BYTES_PER_UNIT = 36          # bytes of fp32 factors read per (row or column) x block-rank (DESIGN.md far-field)
# dram__bytes_read.sum + dram__bytes_write.sum of the k_far launches / their algorithmic factor bytes, from the ncu --set full
# capture summarised in profiles/r02c_far_c3.md (per launch; the bench line scales it to the launches of one step)
FAR_TRAFFIC_RATIO = 1.046
ORACLE_SAMPLE_N = {"c1": 2048, "c2": 8192, "c3": 24576, "c4": 16384, "c5": 16000, "p1": 60000, "p2": 60000}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy read+write)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons every 200 ms during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index, period_ms=200):
        self.index = index
        self.period_ms = int(period_ms)
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", str(self.period_ms)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            f = [t.strip() for t in line.split(",")]
            if len(f) >= 7:
                self.rows.append(f)

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for f in self.rows:
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(value, world, device):
    """max of a per-rank scalar over all ranks (the contract's max-over-ranks timing); no data-path collective exists"""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def make_inputs(workload, rank):
    """seeded synthetic cloud of the named config; replicas (rank > 0) draw their own seed"""
    import synth
    cfg = dict(synth.CONFIGS[workload])
    if cfg["shape"] in ("two_drops", "filament_sphere"):               # the paper's own workloads; one seed
        return synth.config(workload)
    n = cfg["n"]
    if cfg["shape"] == "cube":
        X = synth.cube_cloud(n, cfg["phi"], seed=rank)
    elif cfg["shape"] == "ball":
        X = synth.ball_cloud(n, cfg["phi"], seed=rank)
    else:
        X = synth.chain_cloud(cfg["n_chains"], cfg["n_beads"], cfg["phi"], seed=rank)
    if cfg["forces"] == "gaussian":
        F = synth.gaussian_forces(n, seed=2 + 16 * rank)
    elif cfg["forces"] == "gravity":
        F = synth.gravity_forces(n)
    else:
        import numpy as np
        F = synth.filament_forces(X.astype(np.float64), cfg["n_chains"], cfg["n_beads"]).astype(np.float32)
    return cfg, X, F


def oracle_step_sample(workload, n_sample):
    """One oracle pass (tree + Alg. 1 + Alg. 2 + near + far + three-body, fp64) over an n_sample-particle
    cloud of the workload's recipe; returns (seconds, particles, threads)."""
    import numpy as np
    import synth
    import oracle
    cfg, X, F = synth.config(workload, n=n_sample)
    mlp2 = synth.xavier_mlp(synth.MLP2_DIMS, 1)
    mlp3 = synth.xavier_mlp(synth.MLP3_DIMS, 3)
    oracle.lib()                                                   # compile outside the timed region
    t0 = time.perf_counter()
    H = oracle.HMatrix(X, mlp2, leaf=cfg["leaf"], eta=cfg["eta"], a=1.0)
    U, _ = H.matvec(F, cfg["tol"])
    if cfg["rcut3"] > 0:
        U3, _ = oracle.three_body(X, F, mlp3, cfg["rcut3"])
        U = U + U3
    Xn = oracle.euler(X, U, cfg["dt"])
    dt = time.perf_counter() - t0
    assert np.isfinite(Xn).all()
    return dt, len(X), oracle.num_threads()


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on a bounded sample of the workload, rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    n_s = ORACLE_SAMPLE_N[args.workload]
    import synth
    cfg = synth.CONFIGS[args.workload]
    for _ in range(args.warmup_ref):
        oracle_step_sample(args.workload, n_s)
    ts = []
    cores = 0
    for _ in range(args.steps):
        t, n, cores = oracle_step_sample(args.workload, n_s)
        ts.append(t)
    total = sum(ts)
    v = n_s * len(ts) / total
    sample = ("%d-particle cloud of the same recipe (shape %s, phi %s, leaf %d, eta %.1f, zeta %.0e, rcut3 %.1f), "
              "one full oracle step each" % (n_s, cfg["shape"], cfg["phi"], cfg["leaf"], cfg["eta"], cfg["tol"], cfg["rcut3"]))
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup_ref, "ms_per_step": 1e3 * total / len(ts), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.workload), "sample_particles": n_s},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_name(w, c=None):
    import synth
    c = c or synth.CONFIGS[w]
    src = "BASELINE.json configs[%d]" % (int(w[1]) - 1) if w[0] == "c" else "PAPER.md Sec. 4.3.%s at the paper's parameters, random-init MLPs" % w[1]
    return ("%s: N=%s %s phi=%s, leaf %d, eta=%.1f, zeta=%.0e, rcut3=%.1f, kappa_max=%s, MLP2 4-32-32-9, MLP3 7-64-64-9 (%s)"
            % (w, c["n"], c["shape"], c["phi"], c["leaf"], c["eta"], c["tol"], c["rcut3"], c.get("kappa_max", 0.0) or "inf (plain listing)", src))


def run_gpu(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    import synth
    import paper_2505_08174_b200 as hh

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg, X, F = make_inputs(args.workload, rank)
    for key, val in (("eta", args.eta), ("tol", args.tol), ("leaf", args.leaf), ("kappa_max", args.kappa_max)):
        if val is not None:
            cfg[key] = val                                              # sweeps of config 3 (eta, zeta); otherwise the config's own
    N = len(X)
    mlp2 = synth.xavier_mlp(synth.MLP2_PAPER_DIMS if args.paper_mlp else synth.MLP2_DIMS, 1)
    mlp3 = synth.xavier_mlp(synth.MLP3_DIMS, 3) if cfg["rcut3"] > 0 else None
    free, _ = torch.cuda.mem_get_info(dev)
    ws = int(min(free * 0.85, args.workspace_gb * (1 << 30)))
    ctx = hh.Context(mlp2, mlp3, leaf_size=cfg["leaf"], eta=cfg["eta"], aca_tol=cfg["tol"], rcut3=cfg["rcut3"],
                     kappa_max=float(cfg.get("kappa_max", 0.0)), near_path=args.near_path, aca_precision=args.aca_precision,
                     workspace_bytes=ws, device=dev)
    ctx.enable_timing(True)
    if args.aca_impl:
        ctx.set_aca_impl(args.aca_impl)
    if args.far_impl:
        ctx.set_far_impl(args.far_impl)
    stream = torch.cuda.current_stream(dev)
    Xd = torch.from_numpy(X).to(dev)
    Fd = torch.from_numpy(F).to(dev)
    Ud = torch.empty_like(Fd)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    dt = float(cfg["dt"])

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def harness_forces():
        """multi-step filament workloads: the harness recomputes the internal forces from the current positions (device
        tensors, synth's generator with xp = torch); input generation, outside the timed events"""
        if cfg["forces"] == "filament":
            Fd.copy_(synth.filament_forces(Xd.double(), cfg["n_chains"], cfg["n_beads"], xp=torch).float())
        elif cfg["forces"] == "mixture":
            Fd.copy_(synth.mixture_forces(Xd.double(), cfg["n_chains"], cfg["n_beads"], xp=torch).float())

    def one_step():
        harness_forces()
        flush.fill_(1)                                                  # L2 flush between iterations (outside the events)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        ctx.step(Xd, Fd, Ud, dt=dt)
        e1.record(stream)
        e1.synchronize()
        return e0.elapsed_time(e1), ctx.stats()

    for _ in range(args.warmup):
        one_step()
    barrier()
    clocks = ClockSampler(local, args.clock_period_ms)
    if rank == 0 and args.clock_period_ms > 0:
        clocks.start()
    t_wall = time.perf_counter()
    ms, stats = [], []
    for _ in range(args.steps):
        m, st = one_step()
        ms.append(m)
        stats.append(st)
    barrier()
    t_wall = time.perf_counter() - t_wall
    clk = clocks.stop() if rank == 0 else None
    total_ms = float(sum(ms))
    total_ms = max_over_ranks(total_ms, world, dev)
    assert torch.isfinite(Ud).all().item(), "non-finite velocities"

    # ---- end to end through the public API with HOST buffers (pinned), copies inside the timed region ----
    Xh = torch.from_numpy(X.copy()).pin_memory()
    Fh = torch.from_numpy(F.copy()).pin_memory()
    Uh = torch.empty_like(Fh).pin_memory()
    ke = max(1, min(args.steps, args.e2e_steps))
    ctx.step_host(Xh, Fh, Uh, dt=dt)                                   # warm-up
    barrier()
    t0 = time.perf_counter()
    for _ in range(ke):
        flush.fill_(1)
        ctx.step_host(Xh, Fh, Uh, dt=dt)                                # returns after the D2H copies have completed
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, world, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    K = args.steps
    st = stats[-1]
    mean = lambda k: float(np.mean([s[k] for s in stats]))
    hbm_peak, peak_src = peaks()
    far_bytes = float(st["factor_bytes"])                               # 36 B x sum over blocks of rank x (rows + cols)
    far_ms = mean("ms_far")
    far_gbs = far_bytes / (far_ms * 1e-3) / 1e9 if far_ms > 0 else 0.0
    step_ms = total_ms / K
    stages = {k: mean(k) for k in ("ms_tree", "ms_blocks", "ms_aca", "ms_near", "ms_far", "ms_three", "ms_other")}
    apply_ms = stages["ms_near"] + stages["ms_far"] + stages["ms_three"] + stages["ms_other"]
    line = {
        "metric": METRIC, "value": world * N * K / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(args.workload, cfg), "parallelism": "replicas x%d (no sharding, no collectives)" % world,
                   "l2": "explicit 256 MB flush write between timed iterations; each step also streams its factor arena (>> L2)",
                   "arena_gb": st["arena_bytes"] / 2 ** 30, "aca_batches_per_step": st["aca_batches"],
                   "near_path": "%d (%s)" % (args.near_path, ["fp32 ALU", "tcgen05 tf32 + tanh.approx (2e-3 path)", "tcgen05 split tf32 + tanhf (fp32-class)"][args.near_path]),
                   "mlp2": "4-128-512-128-9 (paper-size hidden layers, tcgen05 tf32 tile, tolerance 2e-3)" if args.paper_mlp else "4-32-32-9",
                   "aca_precision": "%d (%s)" % (args.aca_precision, ["fp32 entries in Alg. 2", "fp64 entries and residuals in Alg. 2 (parity mode)"][args.aca_precision])},
        "clocks": clk,
        "e2e": {"value": world * N * ke / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 24 * N, "d2h_bytes_per_step": 24 * N,
                "steps": ke, "api": "hh_step_host (pinned host X, F in; U, X out)"},
        "gpu_launches": int(sum(s["n_launches"] for s in stats)),
        "stages_ms": stages,
        "apply_only": {"value": N / (apply_ms * 1e-3) if apply_ms > 0 else None, "unit": UNIT,
                       "what": "near + far + three-body + self/permute with factors given (ACA, tree, blocks excluded)"},
        "counts": {k: st[k] for k in ("n_nodes", "n_leaves", "n_admissible", "n_inadmissible", "near_entries", "far_rows_cols",
                                      "sum_rank", "aca_entries", "factor_bytes", "aca_not_converged", "aca_singular", "fallback_entries", "n_faces")},
        "roofline": {"kernel": "k_far (far-field apply U^tau += C (Q F^sigma), all size classes and arena batches of one step)",
                     "bound": "hbm", "achieved": far_gbs, "peak": hbm_peak, "unit": "GB/s", "frac": far_gbs / hbm_peak,
                     "traffic": FAR_TRAFFIC_RATIO * far_bytes if FAR_TRAFFIC_RATIO else None,
                     "traffic_note": "dram bytes of the k_far launches of one step = ncu-measured ratio x algorithmic bytes (profiles/r02c_far_c3.md); not re-collected in this run",
                     "peak_source": peak_src, "share_of_step": far_ms / step_ms,
                     "algorithmic_bytes_per_step": far_bytes, "ms_per_step": far_ms},
        "wall_s_timed_region": t_wall,
    }
    if args.cpu_baseline and world == 1:
        n_s = ORACLE_SAMPLE_N[args.workload]
        t, n, cores = oracle_step_sample(args.workload, n_s)
        line["cpu_baseline"] = {"value": n / t, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "one full oracle step (fp64) on a %d-particle cloud of the same recipe, %.1f s" % (n, t)}
    ctx.close()
    if args.with_c4 and world == 1 and args.workload == "c3":
        # the metric is quoted at 1M AND 10M particles: the 10M point (BASELINE.json configs[3]) rides along as a sub-record
        del ctx, Xd, Fd, Ud, flush
        torch.cuda.empty_cache()
        line["c4"] = sub_record("c4", args, dev, hbm_peak)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def sub_record(workload, args, dev, hbm_peak):
    """one warm-up + one timed hh_step of `workload` on this GPU (the 10M half of the metric beside the 1M line): its own
    ms_per_step, stages, counts and far-field roofline.  Inputs resident in HBM, L2 flushed, CUDA events."""
    import torch
    import synth
    import paper_2505_08174_b200 as hh
    cfg, X, F = make_inputs(workload, 0)
    N = len(X)
    mlp2 = synth.xavier_mlp(synth.MLP2_DIMS, 1)
    mlp3 = synth.xavier_mlp(synth.MLP3_DIMS, 3) if cfg["rcut3"] > 0 else None
    free, _ = torch.cuda.mem_get_info(dev)
    ws = int(min(free * 0.85, args.workspace_gb * (1 << 30)))
    ctx = hh.Context(mlp2, mlp3, leaf_size=cfg["leaf"], eta=cfg["eta"], aca_tol=cfg["tol"], rcut3=cfg["rcut3"],
                     kappa_max=float(cfg.get("kappa_max", 0.0)), near_path=args.near_path, aca_precision=args.aca_precision,
                     workspace_bytes=ws, device=dev)
    ctx.enable_timing(True)
    if args.aca_impl:
        ctx.set_aca_impl(args.aca_impl)
    if args.far_impl:
        ctx.set_far_impl(args.far_impl)
    stream = torch.cuda.current_stream(dev)
    Xd, Fd = torch.from_numpy(X).to(dev), torch.from_numpy(F).to(dev)
    Ud = torch.empty_like(Fd)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ms = None
    for _ in range(2):                                                  # warm-up, then the timed step
        flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        ctx.step(Xd, Fd, Ud, dt=float(cfg["dt"]))
        e1.record(stream)
        e1.synchronize()
        ms = e0.elapsed_time(e1)
    st = ctx.stats()
    assert torch.isfinite(Ud).all().item(), "non-finite velocities"
    far_gbs = st["factor_bytes"] / (st["ms_far"] * 1e-3) / 1e9 if st["ms_far"] > 0 else 0.0
    out = {"workload": workload_name(workload, cfg), "steps": 1, "warmup": 1, "ms_per_step": ms, "value": N / (ms * 1e-3), "unit": UNIT,
           "stages_ms": {k: st[k] for k in ("ms_tree", "ms_blocks", "ms_aca", "ms_near", "ms_far", "ms_three", "ms_other")},
           "counts": {k: st[k] for k in ("n_admissible", "n_inadmissible", "near_entries", "sum_rank", "aca_entries", "factor_bytes", "aca_batches",
                                         "aca_not_converged", "aca_singular")},
           "gpu_launches": int(st["n_launches"]),
           "roofline": {"kernel": "k_far", "bound": "hbm", "achieved": far_gbs, "peak": hbm_peak, "unit": "GB/s", "frac": far_gbs / hbm_peak,
                        "algorithmic_bytes_per_step": float(st["factor_bytes"]), "ms_per_step": st["ms_far"]}}
    ctx.close()
    del ctx, Xd, Fd, Ud, flush
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c3", choices=["c1", "c2", "c3", "c4", "c5", "p1", "p2"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workspace-gb", type=float, default=150.0)
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--eta", type=float, default=None, help="override the config's eta (config 3 sweep)")
    ap.add_argument("--tol", type=float, default=None, help="override the config's ACA tolerance zeta (config 3 sweep)")
    ap.add_argument("--leaf", type=int, default=None)
    ap.add_argument("--kappa-max", type=float, default=None, help="S-18b limit on the pivot-block condition number")
    ap.add_argument("--near-path", type=int, default=2, choices=[0, 1, 2], help="0 fp32 ALU, 1 tcgen05 tf32 + tanh.approx (2e-3), 2 tcgen05 split tf32 + tanhf")
    ap.add_argument("--aca-precision", type=int, default=0, choices=[0, 1], help="1 = fp64 entries and residuals in Alg. 2 (parity mode)")
    ap.add_argument("--aca-impl", type=int, default=0, choices=[0, 1, 2, 3, 4], help="hh_set_aca_impl: 0 lock-step, entries and update in separate launches (default), 1 one CTA per block, 2 lock-step with TMA-staged terms, 3 lock-step, fused, 4 = 0 on two half-batches (update of one beside the entries of the other)")
    ap.add_argument("--far-impl", type=int, default=0, choices=[0, 1, 2], help="hh_set_far_impl: 0 ring kernels for blocks <= 1024 (default), 1 one CTA per block, 2 ring kernel only for blocks <= 256")
    ap.add_argument("--paper-mlp", action="store_true", help="two-body MLP with the paper's hidden layers 128/512/128 (tensor-core tile)")
    ap.add_argument("--clock-period-ms", type=int, default=200, help="nvidia-smi sampling period during the timed region (0 = no sampling: to measure what the sampler itself costs)")
    ap.add_argument("--no-cpu-baseline", dest="cpu_baseline", action="store_false")
    ap.add_argument("--no-c4", dest="with_c4", action="store_false", help="skip the 10M-particle sub-record of the default (c3) run")
    args = ap.parse_args()
    args.warmup_ref = min(args.warmup, 1)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
