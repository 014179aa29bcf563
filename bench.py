#!/usr/bin/env python
"""bench.py -- GNEP hot path (loss + analytic gradient + Adam, one full-batch epoch = one step).

  python bench.py --gpus N --steps K --warmup W [--config C] [--impl reference]

Our arm: the CUDA library through its C ABI (paper_2507_00528_b200.Gnep).  `value` is atom-environments/s
with the batch resident in HBM; `e2e` is the same metric through the C-ABI calls with HOST buffers
(parameters in, loss terms and gradient out, every step).  `roofline` is the dominant kernel against the
plain-FP32 ALU peak (or HBM) and `cpu_baseline` is the fp64 oracle timed on the host cores on a bounded
sample.  --impl reference times the oracle itself (this tier's reference arm).
Inputs are synthetic and seeded (gnep_synth); labels come from a teacher model of the same architecture.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import gnep_synth as gs  # noqa: E402

METRIC = "GNEP atom-envs/s & epoch time (loss+grad+Adam), % of FP32/HBM roofline"
UNIT = "atom-envs/s"
LR = 1e-3


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config index (default 4: throughput scale)")
    ap.add_argument("--structs", type=int, default=0, help="override the number of structures (debugging)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-structs", type=int, default=0, help="structures in the oracle sample (0 = auto)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--minibatch", type=int, default=0,
                    help="structures per mini-batch: time the paper's training regime (P:142: mini-batches of size 1), one "
                         "Adam step per mini-batch through shared handles, instead of the full-batch epoch")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_epoch_time(config, spec, n_structs, steps, warmup):
    """Time the fp64 oracle (as it stands, OpenMP over structures) on the first n_structs structures:
    loss + analytic gradient + Adam per step.  Returns (seconds per step, atoms, threads)."""
    from oracle import gnep_oracle as orc
    sp = orc.make_spec(spec)
    b = gs.make_batch(config, n_structs=n_structs)
    ob = orc.Batch(sp, b["atom_offsets"], b["positions"], b["cells"], b["types"])
    theta = gs.draw_params(spec, config, "student")
    teacher = gs.draw_params(spec, config, "teacher")
    qs = gs.q_scale_from(orc.descriptors(sp, theta, ob))
    E, F, W = gs.add_label_noise(config, b["atom_offsets"], *orc.predict(sp, teacher, qs, ob))
    ob.set_refs(E, F, W)
    m = np.zeros_like(theta); v = np.zeros_like(theta)
    th = theta.copy()
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        _, g = orc.loss_and_grad(sp, th, qs, ob)
        orc.adam_step(th, m, v, g, it + 1, LR)
        if it >= warmup:
            times.append(time.perf_counter() - t0)
    return float(np.mean(times)), int(ob.N), orc.max_threads()


def auto_cpu_structs(config, spec, target_s=12.0):
    """Pick a sample size so that one oracle epoch takes roughly target_s seconds."""
    probe = {0: 4, 1: 4, 2: 4, 3: 6, 4: 4}[config]
    t, n_atoms, _ = oracle_epoch_time(config, spec, probe, 1, 0)
    per_struct = max(t / probe, 1e-6)
    return int(max(probe, min(gs.N_STRUCTS[config], round(target_s / per_struct))))


def run_reference(args):
    """Reference arm of this tier: the oracle on the host cores, bounded sample, same metric/config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    spec = dict(gs.MODEL_SPECS[args.config])
    n_s = args.cpu_structs or auto_cpu_structs(args.config, spec, target_s=max(4.0, 100.0 / max(1, args.steps + args.warmup)))
    sec, n_atoms, threads = oracle_epoch_time(args.config, spec, n_s, args.steps, args.warmup)
    val = n_atoms / sec
    sample = "first %d structures (%d atoms) of %s, one loss+grad+Adam epoch per step" % (n_s, n_atoms, gs.WORKLOAD_NAMES[args.config])
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": gs.WORKLOAD_NAMES[args.config], "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def setup_model(args, rank, world, torch):
    """Create the model, load this rank's shard, derive q_scale, label with the teacher, set the student."""
    from paper_2507_00528_b200 import Gnep
    cfg = args.config
    spec = dict(gs.MODEL_SPECS[cfg])
    S = args.structs or gs.N_STRUCTS[cfg]
    t0 = time.perf_counter()
    b = gs.make_batch(cfg, n_structs=S, first=rank * S, workers=min(16, os.cpu_count() or 1))
    t_gen = time.perf_counter() - t0
    g = Gnep(spec, stream=torch.cuda.current_stream())
    t0 = time.perf_counter()
    g.load_batch(b["atom_offsets"], b["positions"], b["cells"], b["types"])
    torch.cuda.synchronize()
    t_load = time.perf_counter() - t0
    theta = gs.draw_params(spec, cfg, "student").astype(np.float32)
    teacher = gs.draw_params(spec, cfg, "teacher").astype(np.float32)
    g.set_params(theta)
    q = g.descriptors()
    lo, hi = q.min(axis=0).astype(np.float64), q.max(axis=0).astype(np.float64)
    if world > 1:                       # the scaling is a property of the whole job
        import torch.distributed as dist
        tl = torch.tensor(lo, device="cuda"); th = torch.tensor(hi, device="cuda")
        dist.all_reduce(tl, op=dist.ReduceOp.MIN); dist.all_reduce(th, op=dist.ReduceOp.MAX)
        lo, hi = tl.cpu().numpy(), th.cpu().numpy()
    qs = gs.q_scale_from(np.stack([lo, hi]))
    del q
    g.set_q_scale(qs)
    g.set_params(teacher)
    E, F, W = g.predict()
    E, F, W = gs.add_label_noise(cfg, b["atom_offsets"], E, F, W)
    g.set_targets(E, F, W)
    g.set_params(theta)
    info = g.batch_info()
    return g, spec, b, info, theta, dict(gen_s=t_gen, load_batch_s=t_load)


def run_ours(args):
    import torch
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    torch.cuda.set_stream(torch.cuda.Stream())      # the library's work and torch's events share this stream
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    g, spec, b, info, theta0, setup_t = setup_model(args, rank, world, torch)
    N_local = info["n_atoms"]; S_local = info["n_structs"]
    P = g.num_params()
    N_glob, S_glob = N_local, S_local
    grad_t = torch.empty(P, dtype=torch.float32, device="cuda")
    if world > 1:
        from paper_2507_00528_b200 import sharding
        N_glob, S_glob = sharding.setup_sharded(g, dist, N_local, S_local, device="cuda")

    def step_multi():
        sharding.sharded_step(g, dist, grad_t, LR)

    def run_steps(k):
        if world == 1:
            g.train_epochs(k, LR, want_terms=False)
        else:
            for _ in range(k):
                step_multi()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing ----
    run_steps(args.warmup)
    launches0 = g.launch_count()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record()
    run_steps(args.steps)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    launches = g.launch_count() - launches0
    if world > 1:
        t = torch.tensor([ms], device="cuda"); dist.all_reduce(t, op=dist.ReduceOp.MAX); ms = float(t[0])
    ms_step = ms / args.steps
    value = N_glob / (ms_step * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (theta in; loss terms + gradient out) ----
    th_host = torch.from_numpy(g.get_params()).pin_memory()
    grad_host = torch.empty(P, dtype=torch.float32).pin_memory()
    th_np, grad_np = th_host.numpy(), grad_host.numpy()

    def step_e2e():
        g.set_params(th_np)                                         # H2D: P floats
        terms, _ = g.loss_and_grad(want_terms=True, grad=grad_np)  # D2H: P floats + 5 floats
        if world > 1:
            grad_t.copy_(grad_host, non_blocking=True); dist.all_reduce(grad_t); g.set_grad(grad_t)
        g.adam_step(LR)
        g.get_params(th_np)                                         # D2H: P floats (the step's result)
        return terms

    for _ in range(min(2, args.warmup)):
        step_e2e()
    barrier()
    t0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        last_terms = step_e2e()
    e1.record()
    barrier()
    ms_e2e = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3)
    if world > 1:
        t = torch.tensor([ms_e2e], device="cuda"); dist.all_reduce(t, op=dist.ReduceOp.MAX); ms_e2e = float(t[0])
    e2e = {"value": N_glob / (ms_e2e / args.steps * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 4 * P,
           "d2h_bytes_per_step": 8 * P + 20, "what": "gnep_set_params(host) + gnep_loss_and_grad(host terms, host grad) + gnep_adam_step + gnep_get_params(host)"}

    # ---- per-phase device times (CUDA events on the launching stream) and the roofline of the dominant kernel ----
    from paper_2507_00528_b200 import flopmodel as fm
    g.set_profiling(1)
    acc = {}
    nprof = max(3, min(args.steps, 10))
    for _ in range(nprof):
        g.loss_and_grad(want_terms=True)
        g.adam_step(LR)
        for name, t_ms in g.phase_times():
            acc[name] = acc.get(name, 0.0) + t_ms / nprof
    g.set_profiling(0)
    tot_phase = sum(acc.values())
    npr, npa = info["n_pairs_radial"], info["n_pairs_angular"]
    mflops = fm.method_flops(spec, N_local, npr, npa); mbytes = fm.method_bytes(spec, N_local, npr, npa)
    dflops = fm.phase_flops(spec, N_local, npr, npa); dbytes = fm.phase_bytes(spec, N_local, npr, npa)
    if "a1_descriptor_contraction" in acc:     # descriptor pair sweeps hoisted to load time: only the contraction is in the epoch
        cf, cb = fm.contraction_phase(spec, N_local)
        for dct, val in ((mflops, cf), (dflops, cf), (mbytes, cb), (dbytes, cb)):
            dct["a1_descriptor_contraction"] = val
            dct.pop("a1_radial_descriptor", None); dct.pop("a1_angular_descriptor", None)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "measured copy bandwidth (MEASURED_PEAKS.json)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    # FP32 FMA peak measured in this run (register-only FMA chains on every SM, ~60 ms, CUDA events) next to the nominal one
    pk = g.measure_fp32_peak(60.0)
    fp32_meas, fp32_nom = pk["tflops"], fm.fp32_peak_tflops()
    top = max(acc, key=acc.get)
    t_top = acc[top] * 1e-3
    bound = fm.PHASE_BOUND.get(top, "alu")
    # committed ncu capture of this workload, if any: DRAM bytes of the dominant kernel per launch
    traffic, traffic_src, capture = None, None, None
    tfile = os.path.join(ROOT, "profiles", "r2_cfg%d_traffic.csv" % args.config)
    if not args.structs and os.path.exists(tfile):
        for ln in open(tfile):
            f = ln.strip().split(",")
            if f and f[0] == top:
                traffic = int(float(f[-1])); traffic_src = "committed capture profiles/%s (ncu --set full, not re-measured in this run)" % os.path.basename(tfile)
                if len(f) >= 8:     # pipe utilisations of the same capture: what the kernel is really bound by
                    capture = {"fma_pipe_pct": float(f[2]), "issue_slots_pct": float(f[3]), "shared_memory_pipe_pct": float(f[4])}
    if bound == "hbm":
        ach = mbytes[top] / t_top / 1e9
        roof = {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "traffic": traffic,
                "peak_source": hbm_src}
    else:
        ach = mflops[top] / t_top / 1e12
        roof = {"bound": "alu", "achieved": ach, "peak": fp32_meas, "unit": "TFLOP/s", "frac": ach / fp32_meas, "traffic": traffic,
                "peak_source": "FP32 FMA microbenchmark in this run (gnep_measure_fp32_peak, %.0f ms, implied SM clock %.0f MHz)" % (pk["ms"], pk["implied_sm_mhz"]),
                "frac_of_nominal_peak": ach / fp32_nom, "peak_nominal": fp32_nom,
                "peak_nominal_source": "148 SM x 128 FP32 lanes x 2 flop x 1.965 GHz (B200_PROFILING.md unit counts)"}
    roof.update({"kernel": top, "kernel_ms": acc[top], "kernel_share_of_step": acc[top] / tot_phase,
                 "count": "method-algorithmic (SURVEY 8(d).3, flopmodel.method_flops / method_bytes)",
                 "method_flops": mflops[top], "method_bytes": mbytes[top], "design_flops": dflops[top], "design_bytes": dbytes[top],
                 "bound_from": "ncu captures under profiles/ (flopmodel.PHASE_BOUND), not from a comparison of fractions"})
    if traffic_src:
        roof["traffic_source"] = traffic_src
    if capture:
        roof["counters_from_committed_capture"] = capture
    path_tf = sum(mflops.values()) / (ms_step * 1e-3) / 1e12
    path_tf_design = sum(dflops.values()) / (ms_step * 1e-3) / 1e12
    phases = {k: {"ms": round(v, 4), "bound": fm.PHASE_BOUND.get(k),
                  "method_tflops": round(mflops[k] / (v * 1e-3) / 1e12, 3) if v > 0 else None,
                  "method_gbs": round(mbytes[k] / (v * 1e-3) / 1e9, 1) if v > 0 else None,
                  "design_tflops": round(dflops[k] / (v * 1e-3) / 1e12, 3) if v > 0 else None,
                  "design_gbs": round(dbytes[k] / (v * 1e-3) / 1e9, 1) if v > 0 else None} for k, v in acc.items()}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": gs.WORKLOAD_NAMES[args.config], "n_structs_per_gpu": S_local, "n_atoms_per_gpu": N_local,
                   "n_atoms_total": N_glob, "pairs_radial": info["n_pairs_radial"], "pairs_angular": info["n_pairs_angular"],
                   "n_params": P, "parallelism": "structures sharded over %d GPU(s)" % world,
                   "labels": "teacher model via gnep_predict + noise (1 meV/atom, 20 meV/A)",
                   "l2_between_iterations": "inputs larger than L2 (pair lists + per-atom state >> 126 MB)" if N_local > 200000
                   else "inputs smaller than L2 (small parity config)",
                   "step": "gnep_train_epochs: CUDA graph of loss+grad+Adam" if world == 1 else "loss_and_grad + NCCL all-reduce(P floats) + adam",
                   "generate_s": round(setup_t["gen_s"], 2), "load_batch_s": round(setup_t["load_batch_s"], 3)},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roof,
        "path": {"method_tflops": path_tf, "frac_of_fp32_peak_measured": path_tf / fp32_meas, "frac_of_fp32_peak_nominal": path_tf / fp32_nom,
                 "method_flop_per_atom_env": sum(mflops.values()) / max(N_local, 1), "method_bytes_per_atom_env": sum(mbytes.values()) / max(N_local, 1),
                 "design_tflops": path_tf_design, "design_flop_per_atom_env": sum(dflops.values()) / max(N_local, 1),
                 "fp32_peak_measured_tflops": fp32_meas, "fp32_peak_nominal_tflops": fp32_nom, "fp32_peak_implied_sm_mhz": pk["implied_sm_mhz"],
                 "phase_sum_ms": tot_phase},
        "phases": phases,
        "loss_terms_last": [float(x) for x in last_terms],
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_s = args.cpu_structs or auto_cpu_structs(args.config, spec)
        sec, n_at, threads = oracle_epoch_time(args.config, spec, n_s, 1, 0)
        out["cpu_baseline"] = {"value": n_at / sec, "unit": UNIT, "cores": threads, "kind": "oracle",
                               "sample": "first %d structures (%d atoms) of %s, 1 epoch (loss+grad+Adam), %.1f s" % (n_s, n_at, gs.WORKLOAD_NAMES[args.config], sec)}
    g.destroy()
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def run_minibatch(args):
    """The paper's regime (Fig.1 caption: mini-batches of size 1; Eq.17 schedule): every mini-batch is a resident
    batch on a shared handle, a step = one CUDA-graph replay of loss + gradient + Adam at lr(s).  One JSON line in the
    same contract; `ms_per_step` is per mini-batch step."""
    import torch
    from paper_2507_00528_b200 import Gnep, lr_schedule
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_stream(torch.cuda.Stream())
    cfg, B = args.config, args.minibatch
    spec = dict(gs.MODEL_SPECS[cfg])
    nb = max(1, min(64, (args.structs or gs.N_STRUCTS[cfg]) // B))
    b = gs.make_batch(cfg, n_structs=nb * B)
    off = b["atom_offsets"]
    parent = Gnep(spec, stream=torch.cuda.current_stream())
    theta = gs.draw_params(spec, cfg, "student").astype(np.float32)
    teacher = gs.draw_params(spec, cfg, "teacher").astype(np.float32)
    parent.load_batch(off, b["positions"], b["cells"], b["types"])
    parent.set_params(theta)
    qs = gs.q_scale_from(parent.descriptors())
    parent.set_q_scale(qs)
    parent.set_params(teacher)
    E, F, W = gs.add_label_noise(cfg, off, *parent.predict())
    parent.set_params(theta)
    handles, host = [], []
    for k in range(nb):
        lo, hi = k * B, (k + 1) * B
        a0, a1 = off[lo], off[hi]
        h = parent if k == 0 else parent.create_shared()
        arrs = ((off[lo:hi + 1] - a0).astype(np.int32), b["positions"][a0:a1], b["cells"][lo:hi], b["types"][a0:a1],
                E[lo:hi].astype(np.float64), F[a0:a1].astype(np.float64), W[lo:hi].astype(np.float64))
        h.load_batch(*arrs)
        handles.append(h); host.append(arrs)
    n_total = args.warmup + args.steps

    def step(s, want_terms):
        lr = lr_schedule(s, max(1, n_total // 10), n_total, LR, 1e-2 * LR)
        return handles[s % nb].train_epochs(1, lr, want_terms=want_terms)

    for s in range(args.warmup):
        step(s, False)
    sampler = ClockSampler(int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.synchronize()
    sampler.start()
    l0 = sum(h.launch_count() for h in handles)
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record()
    atoms = 0
    for s in range(args.warmup, n_total):
        step(s, False)
        atoms += int(host[s % nb][0][-1])
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    launches = sum(h.launch_count() for h in handles) - l0
    # end to end: the mini-batch arrives from HOST memory every step (neighbour build included), the loss goes back
    t0 = time.perf_counter()
    e0.record()
    atoms2, h2d = 0, 0
    for s in range(args.steps):
        arrs = host[s % nb]
        handles[s % nb].load_batch(*arrs)
        terms = step(s, True)
        atoms2 += int(arrs[0][-1]); h2d += sum(a.nbytes for a in arrs)
    e1.record()
    torch.cuda.synchronize()
    ms2 = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3)
    out = {"metric": METRIC, "value": atoms / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
           "data": "synthetic",
           "config": {"workload": "%s/minibatch-%d" % (gs.WORKLOAD_NAMES[cfg], B), "minibatches_resident": nb,
                      "atoms_per_step": atoms / args.steps, "steps_per_s": args.steps / (ms * 1e-3),
                      "step": "gnep_train_epochs(1) on a shared handle: CUDA graph of loss+grad+Adam at lr(s) (Eq.17)",
                      "regime": "paper P:142 (mini-batch training); launch/latency-bound, no roofline claimed"},
           "clocks": clocks, "gpu_launches": int(launches), "roofline": None,
           "e2e": {"value": atoms2 / (ms2 * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d // args.steps, "d2h_bytes_per_step": 20,
                   "what": "gnep_load_batch(host arrays of the mini-batch, neighbour build) + train step + loss terms to host"},
           "loss_terms_last": [float(x) for x in terms]}
    for h in handles[1:]:
        h.destroy()
    parent.destroy()
    print(json.dumps(out))


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    elif args.minibatch:
        if int(os.environ.get("RANK", "0")) == 0:
            run_minibatch(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
