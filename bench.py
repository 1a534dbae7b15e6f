#!/usr/bin/env python
"""bench.py -- throughput of the MD two-electron-integral hot path on BASELINE.json configs[1].

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--variants]

A step is one pass of the whole hot path (pair setup, Boys, Hermite Coulomb tensor, both
Hermite->AO contractions, solid-harmonic transform, store) over one batch: the 200,000
independent (dd|dd) shell quartets of BASELINE.json configs[1], K = 3 per shell, solid-harmonic
output, seed 0 (+rank).  Prints ONE JSON line.  With N > 1 (torchrun)
every rank runs its own batch (quartets are independent: no data-path collective; weak scaling).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "FP64 % of B200 peak and shell-quartets/s per (la lb|lc ld) class and K"
UNIT = "shell-quartets/s"
NQ = 200_000
FP64_PEAK_DERIVED_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 37.2


def workload(K, rank=0, n=NQ):
    from paper_2405_01834_b200 import workloads as W
    w = W.config2(K=K, n=n)
    if rank:
        w = W.independent_quartets(f"cfg2_dddd_K{K}_r{rank}", (2, 2, 2, 2), (K,) * 4, n, (0.05, 50.0), (-5.0, 5.0), rank)
    return w


def workload_name(K, pure, n=NQ):
    return (f"BASELINE configs[1]: (dd|dd) FP64, K={K} per shell, {n} independent quartets, centers U[-5,5]^3, "
            f"zeta log-uniform [0.05,50], {'solid-harmonic' if pure else 'Cartesian'} output, seed 0")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.lines, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def time_steps(fn, steps, warmup, flush, dist_barrier):
    """W warm-ups, then K steps timed with CUDA events on the launching (current) stream; L2 is
    flushed between steps (outside the events).  Returns the summed device ms over the K steps."""
    import torch
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    dist_barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for e0, e1 in ev:
        flush.fill_(1.0)                      # 256 MiB write > 126 MB L2
        e0.record()
        fn()
        e1.record()
    torch.cuda.synchronize()
    dist_barrier()
    return sum(e0.elapsed_time(e1) for e0, e1 in ev)


def cpu_baseline(K, pure, nsample):
    """The oracle as it stands, on this box's host cores, on the first nsample quartets."""
    import numpy as np
    import oracle
    w = workload(K)
    sel = np.arange(nsample)
    ia, ib, ic, id_ = w.shell_indices(sel)
    oracle.eri4(w.a.astuple(), w.b.astuple(), w.c.astuple(), w.d.astuple(), ia[:8], ib[:8], ic[:8], id_[:8], pure)
    t = time.perf_counter()
    oracle.eri4(w.a.astuple(), w.b.astuple(), w.c.astuple(), w.d.astuple(), ia, ib, ic, id_, pure)
    dt = time.perf_counter() - t
    return {"value": nsample / dt, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
            "sample": f"first {nsample} of the {NQ} quartets, {dt:.1f} s, gcc -O2 OpenMP over quartets"}, dt


def ncu_traffic(variant):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the timed kernel from the committed ncu --set full capture
    of this workload (profiles/traffic.json: {variant: {"bytes": B, "kernel_sources_sha": S}}), or None when the capture
    is older than the kernel sources it describes (the sha is over csrc/fused2*.cuh|cu)."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get(variant)
    except (OSError, ValueError):
        return None
    if not isinstance(t, dict):
        return None
    return t["bytes"] if t.get("kernel_sources_sha") == kernel_sources_sha(variant) else None


def kernel_sources_sha(variant):
    import glob
    import hashlib
    h = hashlib.sha1()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2405_01834_b200", "csrc", f"{variant}*"))):
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    K, pure = 3, True
    nsample = 4000
    vals = []
    for _ in range(args.warmup):
        cpu_baseline(K, pure, 200)
    for _ in range(args.steps):
        cb, dt = cpu_baseline(K, pure, nsample)
        vals.append((cb, dt))
    tot = sum(dt for _, dt in vals)
    v = nsample * len(vals) / tot
    cb = dict(vals[-1][0]); cb["value"] = v
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(vals),
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                      "data": "synthetic", "config": {"workload": workload_name(K, pure), "sample_per_step": nsample},
                      "cpu_baseline": cb,
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def measure_variant(dw, w, K, pure, steps, warmup, flush, barrier):
    from paper_2405_01834_b200 import engine, workloads as W
    out = dw.alloc_out(pure)
    ms = time_steps(lambda: dw.run(pure, out), steps, warmup, flush, barrier)
    flops = W.flops_model(2, 2, 2, 2, K * K, K * K, pure)
    return {"K": K, "pure": pure, "ms_per_step": ms / steps, "quartets_per_s": w.nquartets * steps / (ms * 1e-3),
            "model_flop_per_quartet": flops, "model_tflops": flops * w.nquartets * steps / (ms * 1e-3) / 1e12,
            "variant": VARIANT_NAME.get(engine.md_last_variant(), "?"),
            "launches_per_step": engine.md_last_launch_count(), "out_bytes": out.numel() * 8}



VARIANT_NAME = {1: "generic", 2: "fused", 3: "mma", 4: "fused2", 5: "warp", 6: "hl", 7: "lowl", 8: "eri3s"}


def per_class_cases():
    """Rows of the per-class table the metric asks for ("per (la lb|lc ld) class and K"): BASELINE configs[0..3] at their
    stated sizes.  (name, workload maker, solid output?)."""
    from paper_2405_01834_b200 import workloads as W
    c = [("cfg0 (pp|pp) K=1 cart n=2000", lambda: W.config1(2000), False)]
    for K in (1, 3):
        for pure in (True, False):
            c.append((f"cfg1 (dd|dd) K={K} {'solid' if pure else 'cart'} n=200000", lambda K=K: W.config2(K=K), pure))
    for (la, lb, lX, K) in [(0, 0, 0, 1), (1, 1, 1, 1), (3, 3, 3, 4), (3, 3, 6, 4)]:
        c.append((f"cfg2 ({la}{lb}|{lX}) K={K} solid n=1000000", lambda la=la, lb=lb, lX=lX, K=K: W.config3(la, lb, lX, K=K), True))
    for ls in [(4, 4, 4, 4), (5, 5, 5, 5), (6, 6, 6, 6), (3, 4, 5, 6)]:
        c.append((f"cfg3 ({ls[0]}{ls[1]}|{ls[2]}{ls[3]}) K=1 solid n=20000", lambda ls=ls: W.config4(ls), True))
    return c


def executed_flops():
    """FP64 flop per quartet that the kernels EXECUTE for each per-class case: DFMA x2 + DMUL + DADD thread instructions plus
    512 per DMMA warp instruction, counted by ncu on a reduced batch (profiles/r02_executed_flops.md names the command).
    Counts are per quartet and independent of the batch size; they are only trusted for the kernels they were taken on."""
    try:
        return json.load(open(os.path.join(ROOT, "profiles", "r02_executed_flops.json")))
    except (OSError, ValueError):
        return {}


def measure_case(name, make, pure, steps, warmup, flush, local, hbm, counted):
    import torch
    from paper_2405_01834_b200 import engine
    w = make()
    dw = engine.DeviceWorkload(w)
    out = dw.alloc_out(pure)
    probe = time_steps(lambda: dw.run(pure, out), 1, warmup, flush, lambda: None)
    steps = int(max(steps, min(200, 600.0 / max(probe, 1e-3))))          # at least 0.6 s timed, so that the clocks are sampled
    with ClockSampler(local) as cs:
        ms = time_steps(lambda: dw.run(pure, out), steps, 0, flush, lambda: None) / steps
    used, nl = engine.md_last_variant(), engine.md_last_launch_count()
    fl = w.flops_model(pure)
    nsh = 3 if w.three_center else 4
    in_bytes = sum(8 * (3 + 2 * s.K) for s in (w.a, w.b, w.c) + (() if w.three_center else (w.d,)))
    out_bytes = out.numel() * 8 // w.nquartets
    rate = w.nquartets / (ms * 1e-3)
    tf = fl * rate / 1e12
    gbs = (in_bytes + out_bytes) * rate / 1e9
    row = {"case": name, "n": w.nquartets, "variant": VARIANT_NAME.get(used, str(used)), "launches": nl, "ms": ms,
           "quartets_per_s": rate, "bound": "hbm" if fl / (in_bytes + out_bytes) < FP64_PEAK_DERIVED_TFLOPS * 1e3 / hbm else "alu",
           "model_flop_per_quartet": fl, "model_tflops": tf, "frac_model": tf / FP64_PEAK_DERIVED_TFLOPS,
           "algorithmic_bytes_per_quartet": in_bytes + out_bytes, "hbm_gbs": gbs, "frac_hbm": gbs / hbm, "steps": steps, "clocks": cs.summary()}
    ex = counted.get(name)
    if ex and ex.get("variant") == row["variant"]:
        row["executed_flop_per_quartet"] = ex["flop_per_quartet"]
        row["frac_executed"] = ex["flop_per_quartet"] * rate / 1e12 / FP64_PEAK_DERIVED_TFLOPS
    else:
        row["executed_flop_per_quartet"] = row["frac_executed"] = None
    del dw, out
    torch.cuda.empty_cache()
    return row


def run_case(args):
    """One pass of one per-class case on a reduced batch (for ncu instruction counts): python bench.py --case NAME --count-n N"""
    import torch
    from paper_2405_01834_b200 import build, engine
    build.build()
    torch.cuda.set_device(0)
    engine.md_init()
    for name, make, pure in per_class_cases():
        if name == args.case:
            w = make()
            n = min(args.count_n, w.nquartets)
            import numpy as np
            from paper_2405_01834_b200 import workloads as W
            ia, ib, ic, id_ = w.shell_indices(np.arange(n))
            ww = W.Workload(w.name, w.a.take(ia), w.b.take(ib), w.c.take(ic), None if w.three_center else w.d.take(id_),
                            None, None, np.stack([np.arange(n, dtype=np.int32)] * 2, 1))
            dw = engine.DeviceWorkload(ww)
            out = dw.alloc_out(pure)
            if args.variant:               # the variant AUTO picks at the case's full size, when the reduced batch would pick another
                engine.md_set_variant({v: k for k, v in VARIANT_NAME.items()}[args.variant])
            dw.run(pure, out)
            torch.cuda.synchronize()
            print(json.dumps({"case": name, "n": n, "variant": VARIANT_NAME.get(engine.md_last_variant()),
                              "launches": engine.md_last_launch_count()}))
            return
    raise SystemExit(f"unknown case {args.case!r}")


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2405_01834_b200 import build, engine, sharding, workloads as W

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the engine has no CPU fallback")
    build.build()
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    barrier = (lambda: dist.barrier()) if world > 1 else (lambda: None)
    engine.md_init()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    K, pure = 3, True
    if world > 1:
        # weak scaling: ONE seeded list of world x 200,000 quartets, rank r takes its contiguous shard (no data-path collective)
        wall = workload(K, 0, n=NQ * world)
        lo, hi = sharding.shard_range(wall.nquartets, rank, world)
        ia, ib, ic, id_ = wall.shell_indices(np.arange(lo, hi))
        w = W.Workload(wall.name, wall.a.take(ia), wall.b.take(ib), wall.c.take(ic), wall.d.take(id_), None, None,
                       np.stack([np.arange(hi - lo, dtype=np.int32)] * 2, 1))
        del wall
    else:
        w = workload(K, rank)
    dw = engine.DeviceWorkload(w)
    with ClockSampler(local) as cs:
        head = measure_variant(dw, w, K, pure, args.steps, args.warmup, flush, barrier)
    clocks = cs.summary()
    ms_total = head["ms_per_step"] * args.steps
    ms_total = sharding.max_over_ranks(ms_total, "cuda")
    value = world * w.nquartets * args.steps / (ms_total * 1e-3)

    # end to end: the host-buffer C-ABI call, pinned host memory, copies inside the timed region
    esteps = max(1, min(args.steps, 3))
    host_out = torch.empty(w.nquartets * w.nout(pure), dtype=torch.float64).pin_memory()
    pinned = [torch.as_tensor(x).pin_memory() for s in (w.a, w.b, w.c, w.d) for x in (s.center, s.exps, s.coefs)]
    hq = torch.as_tensor(w.quartet_idx).pin_memory()

    class _S:
        pass
    hs = []
    for i, s in enumerate((w.a, w.b, w.c, w.d)):
        o = _S(); o.l, o.K, o.n = s.l, s.K, s.n
        o.center, o.exps, o.coefs = pinned[3 * i: 3 * i + 3]
        hs.append(o)
    h2d = sum(t.numel() * t.element_size() for t in pinned) + hq.numel() * 4
    d2h = host_out.numel() * 8

    def e2e_step():
        engine.md_eri4_host(hs[0], hs[1], hs[2], hs[3], None, None, hq, w.nquartets, pure, host_out,
                            nbra=w.nbra, nket=w.nket)
    e2e_step(); e2e_step()                                   # two warm-ups: stream-ordered pool growth, page pinning
    torch.cuda.synchronize(); barrier()
    t0 = time.perf_counter()
    for _ in range(esteps):
        e2e_step()
    torch.cuda.synchronize(); barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = sharding.max_over_ranks(e2e_s, "cuda")
    e2e_val = world * w.nquartets * esteps / e2e_s

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(K, pure), "quartets_per_gpu": w.nquartets, "class": "(dd|dd)", "K": K,
                       "output": "solid", "structure": "independent quartets (2 fresh pairs per quartet)",
                       "l2": "256 MiB flush write between timed steps", "kernel_variant": head["variant"]},
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": esteps, "api": "md_eri4_host, pinned host buffers"},
            "gpu_launches": head["launches_per_step"] * args.steps}

    if rank == 0:
        # roofline of the step (one fused kernel, or pair setup + quartet kernel): algorithmic flops of the
        # Table I model over the CUDA-event duration, against the FP64 DFMA peak.
        dfma_tf, _ = engine.md_fp64_peak(0, 0.5)
        dmma_tf, _ = engine.md_fp64_peak(1, 0.3)
        achieved = head["model_tflops"]
        line["roofline"] = {"bound": "alu", "achieved": achieved, "peak": FP64_PEAK_DERIVED_TFLOPS, "unit": "TFLOP/s",
                            "frac": achieved / FP64_PEAK_DERIVED_TFLOPS, "traffic": ncu_traffic(head["variant"]),
                            "frac_is": "Table-I MODEL flops (dense solid-harmonic contraction) over the peak; frac_executed counts what the kernel issues",
                            "frac_executed": None,
                            "peak_source": "derived: 148 SM x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md)",
                            "peak_measured_dfma_loop": dfma_tf, "peak_measured_dmma_m8n8k4_loop": dmma_tf,
                            "frac_of_measured_dfma": achieved / dfma_tf if dfma_tf else None,
                            "algorithmic_flop_per_quartet": head["model_flop_per_quartet"],
                            "kernel": f"md_eri4 step = {head['launches_per_step']} launch(es) of the {head['variant']} kernel",
                            "hbm_gbs_algorithmic": (head["out_bytes"] + h2d) / (head["ms_per_step"] * 1e-3) / 1e9}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
            line["roofline"]["hbm_peak_gbs_measured"] = peaks.get("hbm_gbs")
        except (OSError, ValueError):
            line["roofline"]["hbm_peak_gbs_measured"] = None
        if world == 1:
            cb, _ = cpu_baseline(K, pure, args.cpu_sample)
            line["cpu_baseline"] = cb
            if not args.no_per_class:
                hbm = line["roofline"]["hbm_peak_gbs_measured"] or 6550.0
                counted = executed_flops()
                line["per_class"] = [measure_case(nm, mk, pu, 2, 3, flush, local, hbm, counted) for nm, mk, pu in per_class_cases()]
                head_ex = counted.get("cfg1 (dd|dd) K=3 solid n=200000")
                if head_ex and head_ex.get("variant") == head["variant"]:
                    ex_tf = head_ex["flop_per_quartet"] * value / 1e12
                    line["roofline"]["executed_flop_per_quartet"] = head_ex["flop_per_quartet"]
                    line["roofline"]["achieved_executed"] = ex_tf
                    line["roofline"]["frac_executed"] = ex_tf / FP64_PEAK_DERIVED_TFLOPS
            if args.variants:
                extra = []
                for k2, p2 in ((1, True), (1, False), (3, False)):
                    w2 = workload(k2)
                    dw2 = engine.DeviceWorkload(w2)
                    extra.append(measure_variant(dw2, w2, k2, p2, args.steps, args.warmup, flush, barrier))
                    del dw2
                line["variants"] = [head] + extra
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------------------
# Per-class sweep (every class reports its achieved fraction): python bench.py --sweep NAME
# writes gpurun_out/sweep_NAME.csv; the default run and its one JSON line are unaffected.
# ------------------------------------------------------------------------------------------------------------

def sweep_cases(name):
    from paper_2405_01834_b200 import workloads as W
    cases = []
    if name == "l2":                 # every class served by both fused kernels, K = 1 and K = 3, solid output
        pairs = [(1, 1), (2, 0), (2, 1), (2, 2)]
        for b in pairs:
            for k in pairs:
                for K in (1, 3):
                    n = 100_000 if K == 1 else 20_000
                    cases.append((f"({b[0]}{b[1]}|{k[0]}{k[1]}) K={K}", lambda b=b, k=k, K=K, n=n: W.independent_quartets(
                        "sw", b + k, (K,) * 4, n, (0.05, 50.0), (-5.0, 5.0), W.class_seed("l2", b, k, K)), True,
                        ("fused", "fused2")))
    elif name == "configs":          # the BASELINE.json configs that exist as generators, AUTO variant
        cases.append(("cfg1 (pp|pp) K=1 cart n=2000", lambda: W.config1(2000), False, ("auto",)))
        cases.append(("cfg1-shape (pp|pp) K=1 cart n=1e6", lambda: W.independent_quartets(
            "sw", (1, 1, 1, 1), (1,) * 4, 1_000_000, (0.1, 20.0), (-3.0, 3.0), 0), False, ("auto",)))
        for K in (1, 3):
            for pure in (True, False):
                cases.append((f"cfg2 (dd|dd) K={K} {'solid' if pure else 'cart'}", lambda K=K: W.config2(K=K), pure, ("auto",)))
        for (la, lb, lX) in [(0, 0, 0), (1, 1, 1), (2, 2, 2), (3, 3, 3), (3, 3, 6), (2, 1, 4)]:
            for K in (1, 4):
                cases.append((f"cfg3 ({la}{lb}|{lX}) K={K} solid", lambda la=la, lb=lb, lX=lX, K=K: W.config3(
                    la, lb, lX, K=K, n=200_000), True, ("auto",)))
        for ls in [(3, 3, 3, 3), (4, 4, 4, 4), (5, 5, 5, 5), (6, 6, 6, 6), (3, 4, 5, 6)]:
            cases.append((f"cfg4 ({ls[0]}{ls[1]}|{ls[2]}{ls[3]}) K=1 solid", lambda ls=ls: W.config4(ls, n=20_000), True, ("auto",)))
    elif name == "all":              # sweep 6 of SURVEY.md 8(d): every canonical class, K = 1, config-4 distribution
        pairs = [(a, b) for a in range(7) for b in range(a + 1)]
        for ib, b in enumerate(pairs):
            for k in pairs[: ib + 1]:
                ls = b + k
                nout = 1
                for l in ls:
                    nout *= 2 * l + 1
                n = int(min(200_000, (1 << 30) // (8 * nout)))
                cases.append((f"({b[0]}{b[1]}|{k[0]}{k[1]})", lambda ls=ls, n=n: W.class_sweep(ls, n), True, ("auto",)))
        for b in pairs:
            for lX in range(7):
                nout = (2 * b[0] + 1) * (2 * b[1] + 1) * (2 * lX + 1)
                n = int(min(200_000, (1 << 30) // (8 * nout)))
                cases.append((f"({b[0]}{b[1]}|{lX})", lambda b=b, lX=lX, n=n: W.class_sweep(b + (lX,), n, K=(1, 1, 1),
                                                                                             three_center=True), True, ("auto",)))
    elif name == "paper":            # sweep 7: the paper's Tables IV and V shapes, bra list x ket list products
        def size(ls, Kb, Kk, three):
            nout = 1
            for l in ls:
                nout *= 2 * l + 1
            fl = W.flops_model(ls[0], ls[1], ls[2], 0 if three else ls[3], Kb, Kk, True)
            n = min(1_000_000, (1 << 30) // (8 * nout), int(6e11 / fl))
            return max(8, int(n ** 0.5))
        four = [(l, l, 0, 0) for l in range(1, 7)] + [(l, 0, l, 0) for l in range(1, 7)] + [(l, l, l, l) for l in range(7)]
        for ls in four:
            for Kb, Kk in ((1, 1), (1, 5), (5, 5)):      # the paper sorts the higher contraction onto the ket
                m = size(ls, Kb, Kk, False)
                cases.append((f"[{ls[0]}{ls[1]}|{ls[2]}{ls[3]}] {{{Kb};{Kk}}}", lambda ls=ls, Kb=Kb, Kk=Kk, m=m: W.paper_microbench(
                    ls, Kb, Kk, m, m), True, ("auto",)))
        three = [(0, 0, l) for l in range(1, 7)] + [(l, l, 0) for l in range(1, 7)] + [(l, l, l) for l in range(7)]
        for ls in three:                                 # the paper's [a|cd] {Ka;Kcd} is (cd|a) here: pair first
            for Ka, Kcd in ((1, 1), (1, 5), (5, 5)):
                m = size(ls, Kcd, Ka, True)
                cases.append((f"[{ls[2]}|{ls[0]}{ls[1]}] {{{Ka};{Kcd}}}", lambda ls=ls, Ka=Ka, Kcd=Kcd, m=m: W.paper_microbench(
                    ls, Kcd, Ka, m, m, three_center=True), True, ("auto",)))
    else:
        raise SystemExit(f"unknown sweep {name!r}")
    return cases


def schwarz_factors(engine, W, mol, ta, tb, pairs):
    """Q_ij = sqrt(max_ab |(ab|ab)|) for every pair of one pair type: md_schwarz on the device (csrc/screen.cu)."""
    import numpy as np
    w = W.config5_class(mol, (ta, tb), (ta, tb), pairs, pairs[:1], np.zeros((1, 2), np.int32))
    dw = engine.DeviceWorkload(w)
    return engine.md_schwarz(dw.a, dw.b, dw.bra_idx, True)          # torch CUDA tensor [npairs]


def run_config5(args):
    """BASELINE configs[4]: the synthetic quadruple-zeta molecule.  Schwarz factors with the engine, exact per-class
    counts of surviving quartets, every l <= 4 class timed on a seeded sample, sweep time extrapolated."""
    import numpy as np
    import torch
    from paper_2405_01834_b200 import build, engine, workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the engine has no CPU fallback")
    build.build()
    torch.cuda.set_device(0)
    engine.md_init()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    thr = 1e-12
    mol = W.config5_molecule()
    ptypes = mol.pair_types(4)
    pairs = {pt: mol.pair_list(*pt) for pt in ptypes}
    t0 = time.perf_counter()
    Qd = {pt: schwarz_factors(engine, W, mol, pt[0], pt[1], pairs[pt]) for pt in ptypes}
    torch.cuda.synchronize()
    Q = {pt: q.cpu().numpy() for pt, q in Qd.items()}               # host copies only for drawing the timed samples
    t_schwarz = time.perf_counter() - t0
    vname = VARIANT_NAME
    rows = ["class,Kbra,Kket,pairs_bra,pairs_ket,quartets_passing,sampled,variant,ms,quartets_per_s,model_tflops,"
            "extrapolated_s" + (",measured_full_s,list_s" if args.full else "")]
    full_s, list_s, full_q = 0.0, 0.0, 0
    rng = np.random.default_rng(5)
    tot_q, tot_s, tot_flop = 0, 0.0, 0.0
    name = lambda t: "spdfg"[t[0]] + (str(t[1]) if t[1] > 1 else "")
    for ib, pb in enumerate(ptypes):
        for pk in ptypes[: ib + 1]:
            same = pb == pk
            count, _ = engine.md_quartet_list(Qd[pb], Qd[pk], thr, same=same, capacity=0)   # exact count on the device
            if count == 0:
                continue
            # The timed call sees a random subset of at most 2048 pairs per side and a sample of the surviving quartets
            # among them: pair setup is then amortised over about as many quartets per pair as in the full sweep.
            sb = np.sort(rng.choice(len(pairs[pb]), min(2048, len(pairs[pb])), replace=False))
            sk = sb if same else np.sort(rng.choice(len(pairs[pk]), min(2048, len(pairs[pk])), replace=False))
            qb_s, qk_s = Q[pb][sb], Q[pk][sk]
            avail = W.schwarz_count(qb_s, qk_s, thr, same)
            if avail == 0:                                   # the subset happens to hold no surviving quartet
                sb = np.argsort(-Q[pb])[:2048]; sk = sb if same else np.argsort(-Q[pk])[:2048]
                sb, sk = np.sort(sb), np.sort(sk)
                qb_s, qk_s = Q[pb][sb], Q[pk][sk]
                avail = W.schwarz_count(qb_s, qk_s, thr, same)
            probe = W.schwarz_sample(rng, qb_s, qk_s, thr, min(avail, 2000), same)
            wp = W.config5_class(mol, pb, pk, pairs[pb][sb], pairs[pk][sk], probe)
            dp = engine.DeviceWorkload(wp); op = dp.alloc_out(True)
            ms_p = time_steps(lambda: dp.run(True, op), 1, 1, flush, lambda: None)
            n = int(min(avail, 200_000, max(len(probe), len(probe) * 100.0 / max(ms_p, 1e-3))))   # about 0.1 s
            qs = probe if n <= len(probe) else W.schwarz_sample(rng, qb_s, qk_s, thr, n, same)
            w = W.config5_class(mol, pb, pk, pairs[pb][sb], pairs[pk][sk], qs)
            dw = engine.DeviceWorkload(w); out = dw.alloc_out(True)
            ms = time_steps(lambda: dw.run(True, out), 2, 1, flush, lambda: None) / 2
            rate = len(qs) / (ms * 1e-3)
            fl = w.flops_model(True)
            cls = f"({name(pb[0])}{name(pb[1])}|{name(pk[0])}{name(pk[1])})"
            row = (f"{cls},{pb[0][1] * pb[1][1]},{pk[0][1] * pk[1][1]},{len(pairs[pb])},{len(pairs[pk])},{count},{len(qs)},"
                   f"{vname.get(engine.md_last_variant(), '?')},{ms:.4f},{rate:.4e},{fl * rate / 1e12:.3f},{count / rate:.3f}")
            tot_q += count; tot_s += count / rate; tot_flop += fl * count
            del dw, out, dp, op
            if args.full and max(pb[0][0], pb[1][0], pk[0][0], pk[1][0]) <= args.full_lmax:
                # the class RUN IN FULL: the whole surviving list (built on the device), all pairs of both types, chunks of the
                # list that reuse one output buffer (the integrals are not consumed: this times their evaluation)
                t1 = time.perf_counter()
                nfull, idx = engine.md_quartet_list(Qd[pb], Qd[pk], thr, same=same, capacity=count)
                torch.cuda.synchronize()
                tl = time.perf_counter() - t1
                assert nfull == count
                wf = W.config5_class(mol, pb, pk, pairs[pb], pairs[pk], np.zeros((1, 2), np.int32))
                dwf = engine.DeviceWorkload(wf)
                per = wf.nout(True)
                chunk = int(max(1, min(count, (16 << 30) // (8 * per))))
                outf = torch.empty(chunk * per, dtype=torch.float64, device="cuda")
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for q0 in range(0, count, chunk):
                    m = min(chunk, count - q0)
                    engine.md_eri4(dwf.a, dwf.b, dwf.c, dwf.d, dwf.bra_idx, dwf.ket_idx, idx[q0:q0 + m], m, True, outf,
                                   nbra=len(pairs[pb]), nket=len(pairs[pk]))
                e1.record()
                torch.cuda.synchronize()
                tf = e0.elapsed_time(e1) * 1e-3
                full_s += tf; list_s += tl; full_q += count
                row += f",{tf:.4f},{tl:.4f}"
                del idx, outf, dwf
            elif args.full:
                row += ",,"
            rows.append(row)
    path = os.path.join(ROOT, "gpurun_out", "sweep_config5.csv")
    os.makedirs(os.path.dirname(path), exist_ok=True)
    open(path, "w").write("\n".join(rows) + "\n")
    print(json.dumps({"sweep": "config5", "csv": os.path.relpath(path, ROOT), "classes": len(rows) - 1, "shells": mol.nshells(),
                      "ao_solid": mol.nao(True), "shell_pairs": int(sum(len(p) for p in pairs.values())),
                      "schwarz_threshold": thr, "schwarz_seconds": t_schwarz, "quartets_passing": tot_q,
                      "extrapolated_sweep_seconds": tot_s, "extrapolated_model_tflops": tot_flop / tot_s / 1e12,
                      **({"full_run": {"lmax": args.full_lmax, "quartets": full_q, "measured_seconds": full_s,
                                       "list_seconds": list_s}} if args.full else {}),
                      "note": "per-class rate measured on a seeded sample of the surviving quartets; counts are exact"}))



def e3_serves(ls):
    """Mirror of eri3s_has_class for 4-center classes: one pair with both l <= 3, the other (c s) or small enough for the dense ket table."""
    nc = lambda l: (l + 1) * (l + 2) // 2
    nh = lambda l: (l + 1) * (l + 2) * (l + 3) // 6
    bra_ok = lambda a, b: a <= 3 and b <= 3

    def ket_ok(c, d):
        ncol = nc(c) * nc(d)
        return d == 0 or (ncol <= 36 and nh(c + d) * (ncol + ncol % 2) <= 1536)
    return (bra_ok(ls[0], ls[1]) and ket_ok(ls[2], ls[3])) or (bra_ok(ls[2], ls[3]) and ket_ok(ls[0], ls[1]))


def run_autotune(args):
    """Times every candidate kernel variant on every canonical class (K = 1; K = 2 per shell for classes with all l <= 3) in the
    independent-quartet structure and writes the measured-best table the library's AUTO consults:
    paper_2405_01834_b200/csrc/variant_table.inc (checked in) and gpurun_out/autotune.csv (all timings)."""
    import numpy as np
    import torch
    from paper_2405_01834_b200 import build, engine, workloads as W
    build.build()
    torch.cuda.set_device(0)
    engine.md_init()
    os.environ["MD_NO_TABLE"] = "1"                       # candidates are forced explicitly; AUTO below means the RULES
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    vid = {"rules": 0, "generic": 1, "fused": 2, "mma": 3, "fused2": 4, "warp": 5, "hl": 6, "lowl": 7, "eri3s": 8}
    pairs = [(a, b) for a in range(7) for b in range(a + 1)]
    cases = []
    for ib, b in enumerate(pairs):
        for k in pairs[: ib + 1]:
            cases.append((b + k, False))
    for b in pairs:
        for lX in range(7):
            cases.append((b + (lX,), True))
    rows = ["class,three_center,contracted,n,variant_asked,variant_used,ms,quartets_per_s"]
    table = []
    with ClockSampler(0) as cs:
        for ls, three in cases:
            lmax = max(ls)
            for contracted in ((False, True) if lmax <= 3 else (False,)):
                nout = 1
                for l in ls:
                    nout *= 2 * l + 1
                fl = W.flops_model(ls[0], ls[1], ls[2], 0 if three else ls[3], 4 if contracted else 1,
                                   (2 if three else 4) if contracted else 1, True)
                n = int(max(296, min(100_000, (1 << 28) // (8 * nout), 4e10 / fl)))
                K = tuple((2 if contracted else 1) for _ in ls)
                w = W.independent_quartets("at", ls, K, n, (0.3, 10.0), (-4.0, 4.0), W.class_seed("at", ls, contracted), three_center=three)
                if lmax <= 1:
                    cands = ["lowl", "fused", "fused2"]
                elif lmax <= 2 and not three:
                    cands = ["fused", "fused2"]
                elif three and max(ls[0], ls[1]) <= 3:
                    cands = ["eri3s", "warp", "mma", "hl"] if lmax > 2 else ["eri3s", "fused", "fused2"]
                else:
                    cands = ["warp", "mma", "hl"]
                if not three and lmax >= 2 and e3_serves(ls):
                    cands = cands + ["eri3s"]            # the one-warp kernel with a two-centre ket (csrc/eri3s_inst.cu: eri3s_has_class)
                dw = engine.DeviceWorkload(w); out = dw.alloc_out(True)
                best = None
                seen = set()
                for c in cands:
                    engine.md_set_variant(vid[c])
                    try:
                        ms = time_steps(lambda: dw.run(True, out), 2, 2, flush, lambda: None) / 2
                        used = VARIANT_NAME.get(engine.md_last_variant(), "?")
                    except engine.MDError as e:
                        rows.append(f"{ls},{int(three)},{int(contracted)},{n},{c},error{e.code},,")
                        continue
                    finally:
                        engine.md_set_variant(0)
                    rows.append(f"{'-'.join(map(str, ls))},{int(three)},{int(contracted)},{n},{c},{used},{ms:.4f},{n / (ms * 1e-3):.4e}")
                    if used in seen:
                        continue                          # the forced variant fell through to one already timed
                    seen.add(used)
                    if best is None or ms < best[0]:
                        best = (ms, used)
                if best:
                    l4 = tuple(ls) + ((0,) if three else ())
                    table.append((l4, three, contracted, best[1]))
                del dw, out
    ck = cs.summary()
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    open(os.path.join(ROOT, "gpurun_out", "autotune.csv"), "w").write("\n".join(rows) + "\n")
    inc = ["// generated by `python bench.py --sweep autotune` (profiles/r02_autotune.md); {la, lb, lc, ld, three-center, contracted, variant}"]
    for l4, three, contracted, v in table:
        inc.append(f"    {{{l4[0]}, {l4[1]}, {l4[2]}, {l4[3]}, {int(three)}, {int(contracted)}, {vid[v]}}},   // {v}")
    open(os.path.join(ROOT, "gpurun_out", "variant_table.inc"), "w").write("\n".join(inc) + "\n")
    print(json.dumps({"sweep": "autotune", "classes": len(table), "timings": len(rows) - 1, "clocks": ck,
                      "table": "gpurun_out/variant_table.inc", "csv": "gpurun_out/autotune.csv"}))


def run_sweep(args):
    if args.sweep == "autotune":
        return run_autotune(args)
    if args.sweep == "config5":
        return run_config5(args)
    import numpy as np
    import torch
    from paper_2405_01834_b200 import build, engine, workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the engine has no CPU fallback")
    build.build()
    torch.cuda.set_device(0)
    engine.md_init()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    vid = {"auto": engine.VARIANT_AUTO, "generic": engine.VARIANT_GENERIC, "fused": engine.VARIANT_FUSED,
           "mma": engine.VARIANT_MMA, "fused2": engine.VARIANT_FUSED2, "warp": engine.VARIANT_WARP, "hl": engine.VARIANT_HL, "lowl": engine.VARIANT_LOWL, "eri3s": engine.VARIANT_ERI3S}
    vname = VARIANT_NAME
    try:
        hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("hbm_gbs", 6550.0)
    except (OSError, ValueError):
        hbm = 6650.0
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    path = os.path.join(ROOT, "gpurun_out", f"sweep_{args.sweep}.csv")
    rows = ["case,n,variant_asked,variant_used,launches,ms,quartets_per_s,model_flop_per_quartet,model_tflops,"
            "frac_fp64_peak,out_gbs,frac_hbm,sm_mhz,throttle_reasons"]
    for label, make, pure, variants in sweep_cases(args.sweep):
        w = make()
        for v in variants:
            engine.md_set_variant(vid[v])
            try:
                ww = w
                if w.nquartets > 2000 and w.quartet_idx is not None:   # bound the time per case: probe on 1000 quartets first
                    sel = np.arange(1000)
                    probe = W.Workload("probe", w.a.take(w.shell_indices(sel)[0]), w.b.take(w.shell_indices(sel)[1]),
                                       w.c.take(w.shell_indices(sel)[2]),
                                       None if w.three_center else w.d.take(w.shell_indices(sel)[3]), None, None,
                                       np.stack([np.arange(1000, dtype=np.int32)] * 2, 1))
                    dp = engine.DeviceWorkload(probe); op = dp.alloc_out(pure)
                    ms_p = time_steps(lambda: dp.run(pure, op), 2, 2, flush, lambda: None) / 2
                    cap = int(max(2000, min(w.nquartets, 1000 * (100.0 if args.sweep == 'all' else 400.0) / max(ms_p, 1e-3))))   # about 0.4 s per step (0.1 s in the 602-class sweep)
                    if cap < w.nquartets:
                        sel = np.arange(cap)
                        ia, ib, ic, id_ = w.shell_indices(sel)
                        ww = W.Workload(w.name, w.a.take(ia), w.b.take(ib), w.c.take(ic),
                                        None if w.three_center else w.d.take(id_), None, None,
                                        np.stack([np.arange(cap, dtype=np.int32)] * 2, 1))
                dw = engine.DeviceWorkload(ww); out = dw.alloc_out(pure)
                with ClockSampler(0) as cs:
                    ms = time_steps(lambda: dw.run(pure, out), args.steps, args.warmup, flush, lambda: None) / args.steps
                ck = cs.summary()
                used, nl = engine.md_last_variant(), engine.md_last_launch_count()
                fl = ww.flops_model(pure)
                tf = fl * ww.nquartets / (ms * 1e-3) / 1e12
                gbs = out.numel() * 8 / (ms * 1e-3) / 1e9
                rows.append(f"{label},{ww.nquartets},{v},{vname.get(used, used)},{nl},{ms:.4f},{ww.nquartets / (ms * 1e-3):.4e},"
                            f"{fl},{tf:.3f},{tf / FP64_PEAK_DERIVED_TFLOPS:.4f},{gbs:.1f},{gbs / hbm:.4f},{ck['sm_mhz']},{'+'.join(ck['reasons']) or 'none'}")
                print(rows[-1], flush=True)
                del dw, out
            finally:
                engine.md_set_variant(engine.VARIANT_AUTO)
    open(path, "w").write("\n".join(rows) + "\n")
    print(json.dumps({"sweep": args.sweep, "csv": os.path.relpath(path, ROOT), "cases": len(rows) - 1}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--variants", action="store_true", help="also time K=1 and Cartesian output")
    ap.add_argument("--cpu-sample", type=int, default=8000)
    ap.add_argument("--no-per-class", action="store_true", help="headline only (skip the per-class table)")
    ap.add_argument("--full", action="store_true", help="--sweep config5: also RUN every class with all l <= --full-lmax in full")
    ap.add_argument("--full-lmax", type=int, default=4)
    ap.add_argument("--case", default=None, help="run ONE per-class case once on --count-n quartets (for ncu instruction counts)")
    ap.add_argument("--count-n", type=int, default=2000)
    ap.add_argument("--variant", default=None, help="with --case: force this kernel variant (generic|fused|mma|fused2|warp|hl)")
    ap.add_argument("--sweep", default=None, help="per-class table instead of the headline: l2 | configs | config5 | all | paper")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and not args.sweep and not args.case:
        # started without a launcher: re-execute under torchrun, one rank per GPU (NCCL's INFO log stays on for rank 0)
        env = dict(os.environ, NCCL_DEBUG=os.environ.get("NCCL_DEBUG", "INFO"))
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", os.environ.get("MASTER_PORT", "29511"), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd, env=env))
    if args.case:
        run_case(args)
    elif args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
