#!/usr/bin/env python
"""bench.py -- throughput of the PIMD/Langevin BAOAB hot path (BASELINE.json metric).

    python bench.py --gpus 1 --steps 20 --warmup 5            # this build (CUDA, sm_100a)
    python bench.py --impl reference --steps 3 --warmup 1     # the oracle on the host cores
    torchrun ... bench.py --gpus N ...                        # N independent replicas ("replicas only")

A step = one pass of the whole hot path (integrator + force evaluation) over the
configs[2] workload (1536 atoms x 32 beads, seeded synthetic water box, random-init se_e2_a weights).
Prints ONE JSON line (rank 0).  See DESIGN.md section 8 for the roofline arithmetic.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "bead-atom-steps/s"
# dram__bytes_read.sum + dram__bytes_write.sum per launch come from the committed `ncu --set full` capture of THIS build
# (profiles/r2_dram_bytes.csv, written from the .ncu-rep as profiles/r2_README.md says); bench.py only reads the file.
DRAM_CSV = os.path.join(ROOT, "profiles", "r2_dram_bytes.csv")
PHASE_KERNEL = {"embed_fwd": "embed_fwd_tc_kernel", "embed_bwd": "embed_bwd_tc_kernel"}


def ncu_dram_bytes(kernel, workload):
    """(read + write bytes per launch, source) of `kernel` at `workload` from the committed capture, or (None, why)."""
    if not os.path.exists(DRAM_CSV):
        return None, "no capture committed"
    import csv
    for row in csv.DictReader(l for l in open(DRAM_CSV) if not l.startswith("#")):
        if row["kernel"] == kernel and row["workload"] == workload:
            return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]), os.path.relpath(DRAM_CSV, ROOT)
    return None, "kernel not in " + os.path.relpath(DRAM_CSV, ROOT)


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sustained=d.get("bf16_tflops_sustained"),
                    sm_max_mhz=d.get("sm_max_mhz", 1965.0), src="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, sm_max_mhz=1965.0, src="fallback")


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.samples, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [l for (t, l) in self.samples if t0 <= t <= t1] or [l for (_, l) in self.samples[-3:]]
        for line in rows:
            p = [q.strip() for q in line.split(",")]
            try:
                sm.append(float(p[0]))
                smax = float(p[1])
            except Exception:
                continue
            for n, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def measure_tf32_peak(seconds=2.0, n=8192):
    """Dense TF32 tensor peak of this GPU, measured the way MEASURED_PEAKS.json measured BF16: torch.matmul (cuBLAS,
    TF32 enabled) on n^3, best of 10 (burst) and back to back for `seconds` (sustained, under the power cap).  Used
    only as the roofline denominator of the kind::tf32 kernels; runs outside every timed region."""
    import torch
    old = torch.backends.cuda.matmul.allow_tf32
    torch.backends.cuda.matmul.allow_tf32 = True
    try:
        a = torch.randn(n, n, device="cuda", dtype=torch.float32)
        b = torch.randn(n, n, device="cuda", dtype=torch.float32)
        c = torch.empty_like(a)
        for _ in range(3):
            torch.matmul(a, b, out=c)
        torch.cuda.synchronize()
        best = 1e30
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(10):
            e0.record(); torch.matmul(a, b, out=c); e1.record(); torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        reps = max(10, int(seconds * 1e3 / best))
        e0.record()
        for _ in range(reps):
            torch.matmul(a, b, out=c)
        e1.record(); torch.cuda.synchronize()
        sus = e0.elapsed_time(e1) / reps
        fl = 2.0 * n ** 3 / 1e12
        return {"tf32": fl / (best * 1e-3), "tf32_sustained": fl / (sus * 1e-3)}
    finally:
        torch.backends.cuda.matmul.allow_tf32 = old
        del a, b, c
        torch.cuda.empty_cache()


def max_over_ranks(value, world, device):
    """Whole-job time = the slowest rank's (replicas only: no data-path collective)."""
    if world <= 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank, world, ms_max):
    """bead-atom-steps/s of the whole job: every rank advanced its own replica by `units_per_rank`."""
    return world * units_per_rank / (ms_max * 1e-3)


def _dist():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# ------------------------------------------------------------------------------------------------
# reference arm = the oracle, as it stands, on the host cores
# ------------------------------------------------------------------------------------------------
def _oracle_sample(cfg_idx, steps, warmup, n_sample_beads):
    """Times `steps` oracle steps (after `warmup`) on a bounded sample: the full box and ring of configs
    [cfg_idx] with the FORCE evaluation restricted to `n_sample_beads` beads (OraclePIMD.only_beads);
    units = sampled beads x atoms x steps."""
    from oracle.pimd import OraclePIMD
    cfg, wb, desc, w = workloads.make_config(cfg_idx)
    orc = OraclePIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=0)
    orc.only_beads = list(range(n_sample_beads))
    if "p_ext_bar" in cfg:
        orc.set_barostat(cfg["p_ext_bar"], cfg["tau_p"])
    orc.set_state(wb["x"], wb["p"])
    orc.set_model(desc, w)
    for _ in range(warmup):
        orc.step(1)
    t0 = time.perf_counter()
    for _ in range(steps):
        orc.step(1)
    dt = time.perf_counter() - t0
    units = n_sample_beads * orc.N * steps
    return units / dt, dt / steps, orc.N, cfg["P"]


def _cores_used():
    try:
        import threadpoolctl
        n = max([p["num_threads"] for p in threadpoolctl.threadpool_info()] + [1])
        return int(n)
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank, world, _ = _dist()
    if rank != 0:
        return 0
    value, s_per_step, N, P = _oracle_sample(args.config, args.steps, args.warmup, 1)
    cores = _cores_used()
    sample = ("configs[%d] box and ring (%d atoms x %d beads); each step = full FP64 integrator + the force "
              "evaluation of 1 of the %d beads (%d bead-atoms)" % (args.config, N, P, P, N))
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": s_per_step * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workloads.CONFIGS[args.config]["name"], "atoms": N, "beads": P, "sample": sample},
        "cpu_baseline": {"value": value, "unit": METRIC, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))
    return 0


# ------------------------------------------------------------------------------------------------
# this build
# ------------------------------------------------------------------------------------------------
def algorithmic_work(counts, N, P):
    """SURVEY 8(d) per-unit figures: useful flops of each force kernel per step."""
    rows = int(counts.sum())
    PN = N * P
    # tensor-eligible work exactly as SURVEY 8(d) counts it: 1250 + 5000 MAC per row and direction for the embedding
    # net, 384,000 + 2 x 57,600 MAC per bead-atom and direction for the fitting net (203 Gflop per step at configs[2])
    flops = {
        "embed_fwd": 2.0 * rows * 6250,
        "embed_bwd": 2.0 * rows * 6250,
        "fitting": 2.0 * PN * 2 * (1600 * 240 + 2 * 240 * 240),
    }
    # "other arithmetic" of 8(d), NOT in any roofline fraction: layer 1, G (x) R and its two backward products, D, dT
    other = {
        "embed_fwd": 2.0 * rows * (25 + 400),
        "embed_bwd": 2.0 * rows * (25 + 400 + 400 + 100),
        "fitting": 2.0 * PN * (1600 * 4 + 2 * 1600 * 4),
    }
    return rows, flops, other


def run_ours(args):
    import torch
    import paper_2602_13553_b200 as pk
    pk.lib()                                        # fail loudly if the CUDA library is missing
    rank, world, local = _dist()
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        torch.cuda.set_device(0)
    peaks = _peaks()
    if rank == 0 and not args.no_tf32_peak:
        peaks.update(measure_tf32_peak())

    cfg, wb, desc, w = workloads.make_config(args.config)
    P, N = cfg["P"], wb["types"].size
    # replicas only (north_star: one GPU, no sharding): every rank advances its own copy with its own seed
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], P, cfg["T"], cfg["dt"], cfg["gamma"], seed=1000 + rank,
                  model_desc=desc)
    x_host = torch.from_numpy(wb["x"]).pin_memory()
    p_host = torch.from_numpy(wb["p"]).pin_memory()
    x_dev, p_dev = x_host.cuda(non_blocking=True), p_host.cuda(non_blocking=True)
    sim.set_model(w)
    sim.set_state(x_dev, p_dev)                     # inputs resident in HBM before the timed region
    if args.compressed:
        sim.set_compressed(True)
        args.no_compressed_leg = True
    if "p_ext_bar" in cfg:                          # configs[4]: NpT, isotropic BZP barostat
        sim.set_barostat(cfg["p_ext_bar"], cfg["tau_p"])

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: K steps ----
    for _ in range(args.warmup):
        sim.step(1)
    launches0 = pk.pimd_get_launch_count(sim.ctx)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # The synthetic workload has no binding potential (random-init weights, forces ~1e-4 eV/A): its atoms drift freely
    # and after ~200 steps two of them overlap (r < 0.01 A), which the library reports as PIMD_ECONTACT.  Long runs are
    # therefore cut into chunks of at most CHUNK steps, each restarted (untimed) from the initial configuration.
    CHUNK = 100

    def timed_steps(n_total):
        ms_sum, done = 0.0, 0
        while done < n_total:
            n = min(CHUNK, n_total - done)
            if done > 0:
                sim.set_state(x_dev, p_dev)
                barrier()
            ev0.record()
            sim.step(n)                             # ONE pimd_step(n) call: n whole steps, no host round trip inside
            ev1.record()
            barrier()
            ms_sum += ev0.elapsed_time(ev1)
            done += n
        return ms_sum

    t_wall0 = time.time()
    ms = timed_steps(args.steps)
    t_wall1 = time.time()
    launches = pk.pimd_get_launch_count(sim.ctx) - launches0
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    ms = max_over_ranks(ms, world, "cuda")
    value = job_throughput(P * N * args.steps, world, ms)

    # ---- per-phase device times (CUDA events on the library's stream) ----
    sim.set_state(x_dev, p_dev)
    pk.pimd_set_profiling(sim.ctx, 1)
    sim.step(max(3, min(10, args.steps)))
    phase = pk.pimd_get_phase_ms(sim.ctx)
    pk.pimd_set_profiling(sim.ctx, 0)
    counts = pk.pimd_get_neighbor_counts(sim.ctx, P, N, 2)
    rows, flops, other = algorithmic_work(counts, N, P)
    names = ["integrator", "neighbour_env", "embed_fwd", "fitting", "embed_bwd"]
    phases = {n: float(phase[q]) for q, n in enumerate(names)}
    dom = max(("embed_fwd", "fitting", "embed_bwd"), key=lambda n: phases[n])
    # tensor roofline.  The embedding kernels and the whole fitting chain (l1_desc, fit_mid, dd_dt) run as three-pass
    # FP16-split kind::f16 tcgen05.mma; only the round-1 chain kept as A/B partner (PIMD_FIT_OLD=1) runs its four
    # 240 x 240 GEMMs as 3xTF32 kind::tf32.  Peaks: FP16 dense = the measured BF16 cuBLAS figure (same tensor rate;
    # sustained: these kernels are timed inside a long step), TF32 dense = measured in this run, else 1/2 of it.
    PN = P * N
    f16_peak = peaks["bf16_sustained"] or peaks["bf16"]
    tf32_peak = peaks.get("tf32_sustained") or 0.5 * f16_peak      # measured in this run; else the guide's nominal 1/2
    mufu_peak = 148 * 16 * peaks["sm_max_mhz"] * 1e6 / 1e12                         # T MUFU op/s
    emb_issue = 2.0 * rows * 3 * (32 * 64 + 64 * 112)                               # K2 x N2 + K3 x N3 of embedding_tc.cu, 3 passes
    issued = {   # (flops issued on padded tiles incl. the 3 passes, peak of that dtype)
        "embed_fwd": [(emb_issue, f16_peak)],
        "embed_bwd": [(2.0 * emb_issue, f16_peak)],                                 # value + derivative rows
        "fitting": ([(3 * 2.0 * PN * (1600 * 240 + 256 * 1600), f16_peak),          # round-1 chain: l1_desc, dd_dt (K padded to 256)
                     (3 * 2.0 * PN * 4 * 240 * 240, tf32_peak)] if os.environ.get("PIMD_FIT_OLD") else
                    [(3 * 2.0 * PN * (2 * 1600 * 240 + 4 * 240 * 240), f16_peak)]),  # l1_desc, dd_dt, the four products of fit_mid
    }
    mufu_ops = {"embed_fwd": 2.0 * rows * 182, "embed_bwd": 2.0 * rows * 182, "fitting": 0.0}   # incl. padded channels
    dom_peak = f16_peak
    achieved = flops[dom] / (phases[dom] * 1e-3) / 1e12
    dom_issued = sum(f for f, _ in issued[dom]) / (phases[dom] * 1e-3) / 1e12
    traffic, traffic_src = ncu_dram_bytes(PHASE_KERNEL.get(dom, dom), cfg["name"])
    roofline = {"kernel": dom, "bound": "tensor", "achieved": achieved, "peak": dom_peak, "unit": "TFLOP/s",
                "frac": achieved / dom_peak, "traffic": traffic, "traffic_src": traffic_src,
                "issued_tflops": dom_issued, "other_arithmetic_gflop": other[dom] / 1e9,
                "note": "achieved = USEFUL tensor-eligible flops exactly as SURVEY 8(d) counts them (6250 MAC per row and "
                        "direction: no recompute, no extra hi/lo passes, no padding, no 'other arithmetic') / live "
                        "CUDA-event time of the phase; peak = FP16 dense = %s BF16 %.0f TFLOP/s (kind::f16 runs at the "
                        "BF16 rate); issued_tflops counts the 3 passes on padded tiles" % (
                            "measured sustained" if peaks["bf16_sustained"] else "measured burst", f16_peak)}
    kernels = {}
    for n in ("embed_fwd", "fitting", "embed_bwd"):
        sec = phases[n] * 1e-3
        t_at_peak = sum(f / (pk_ * 1e12) for f, pk_ in issued[n])
        kernels[n] = {"ms": phases[n], "useful_tflops": flops[n] / sec / 1e12,
                      "issued_tflops": sum(f for f, _ in issued[n]) / sec / 1e12,
                      "frac_tensor_peak_issued": t_at_peak / sec,
                      "frac_tensor_peak_useful": flops[n] / sec / 1e12 / (f16_peak if n != "fitting" else f16_peak)}
        if mufu_ops[n]:
            kernels[n]["frac_mufu_peak"] = mufu_ops[n] / sec / 1e12 / mufu_peak
    kernels["integrator"] = {"ms": phases["integrator"], "algorithmic_GBs": 120.0 * P * N / (phases["integrator"] * 1e-3) / 1e9,
                             "note": "L2-resident at this size (5.9 MB/step); includes 3 memsets"}
    kernels["neighbour_env"] = {"ms": phases["neighbour_env"]}

    # ---- sustained leg: back-to-back steps for seconds, with the clock record (the K-step region above is a burst) ----
    sustained = None
    if args.sustain_s > 0:
        per = max(1, int(0.25 / (ms / args.steps * 1e-3)))                  # steps per call: ~0.25 s of device time
        sampler2 = ClockSampler(local)
        if rank == 0:
            sampler2.start()
            time.sleep(0.25)
        barrier()
        tw0 = time.time()
        n_sus, ms_sus, per = 0, 0.0, min(per, CHUNK)
        while time.time() - tw0 < args.sustain_s:
            sim.set_state(x_dev, p_dev)             # restart (see CHUNK above); its one force evaluation is not timed
            torch.cuda.synchronize()
            ev0.record()
            sim.step(per)
            ev1.record()
            torch.cuda.synchronize()
            ms_sus += ev0.elapsed_time(ev1)
            n_sus += per
        barrier()
        tw1 = time.time()
        ms_sus = max_over_ranks(ms_sus, world, "cuda")
        sustained = {"value": job_throughput(P * N * n_sus, world, ms_sus), "unit": METRIC, "steps": n_sus,
                     "seconds": ms_sus * 1e-3, "ms_per_step": ms_sus / n_sus,
                     "clocks": sampler2.stop(tw0, tw1) if rank == 0 else None}

    # ---- the paper's own model variant: compressed (tabulated) embedding, SURVEY 8(f) NEXT-3 ----
    compressed = None
    if not args.no_compressed_leg:
        # Fresh state: the synthetic workload has no binding potential (random-init weights), so after the ~10^3 steps of
        # the legs above atoms have drifted through each other and some pair sits closer than 0.5 A -- outside the
        # table, which R-28 makes an error (PIMD_ETABLE_RANGE; pimd_step rolls the call back).  The leg therefore starts
        # from the initial configuration again and halves its step count if a ring polymer still reaches r < 0.5 A.
        sim.set_state(x_dev, p_dev)
        sim.set_compressed(True)

        def guarded(n):
            while n >= 1:
                try:
                    sim.step(n)
                    return n
                except pk.PimdError as e:
                    if e.code != pk.PIMD_ETABLE_RANGE:
                        raise
                    n //= 2
            return 0

        guarded(3)
        barrier()
        ev0.record()
        k_c = guarded(args.steps)
        ev1.record()
        barrier()
        # a retry leaves the failed (rolled-back) attempt inside the event pair: time the successful count again, cleanly
        if k_c != args.steps and k_c > 0:
            sim.set_state(x_dev, p_dev)
            barrier()
            ev0.record()
            k_c = guarded(k_c)
            ev1.record()
            barrier()
        ms_c = max_over_ranks(ev0.elapsed_time(ev1), world, "cuda") * (args.steps / max(k_c, 1))
        sim.set_state(x_dev, p_dev)
        pk.pimd_set_profiling(sim.ctx, 1)
        guarded(3)
        ph_c = pk.pimd_get_phase_ms(sim.ctx)
        pk.pimd_set_profiling(sim.ctx, 0)
        sim.set_compressed(False)
        # moments x table products as dense GEMMs: 480 x 100 x 4 MAC per bead-atom and direction
        cmp_flops = 2.0 * PN * 480 * 100 * 4
        compressed = {
            "value": job_throughput(P * N * args.steps, world, ms_c), "unit": METRIC, "ms_per_step": ms_c / args.steps,
            "steps_timed": k_c,
            "speedup_vs_mlp_embedding": (ms / args.steps) / (ms_c / args.steps),
            "phases_ms": {"integrator": float(ph_c[0]), "neighbour_env": float(ph_c[1]), "cmp_fwd": float(ph_c[2]),
                          "fitting": float(ph_c[3]), "cmp_bwd": float(ph_c[4])},
            "cmp_fwd": {"ms": float(ph_c[2]), "bound": "alu (FP32 moment accumulation: shared-memory read-modify-write chain); "
                        "the 480x100x4 products per centre run on tcgen05 from tensor-memory-resident tables",
                        "dense_tflops": cmp_flops / (float(ph_c[2]) * 1e-3) / 1e12,
                        "row_rate_G_per_s": rows / (float(ph_c[2]) * 1e-3) / 1e9},
            "cmp_bwd": {"ms": float(ph_c[4]), "bound": "latency (per tile: dT operand -> 4 M tiles of MMAs -> Q to shared memory -> rows)",
                        "dense_tflops": cmp_flops / (float(ph_c[4]) * 1e-3) / 1e12,
                        "row_rate_G_per_s": rows / (float(ph_c[4]) * 1e-3) / 1e9},
            "note": "same workload with pimd_set_embedding_compressed(1): the model variant the paper's timings use "
                    "(PAPER.md:L76); an approximation of the MLP model (DESIGN R-28), parity against the oracle's compressed "
                    "model in tests/test_gpu_compress.py; the headline `value` above is the MLP path north_star names",
        }

    # ---- integrator alone at HBM-bound size (stand-alone leg, harmonic model) ----
    integ = None
    if rank == 0 and not args.no_integrator_leg:
        integ = integrator_leg(pk, peaks)

    # ---- end to end through the C ABI with host buffers ----
    f_host = torch.empty_like(x_host).pin_memory()
    sim.set_state(x_dev, p_dev)                     # fresh configuration (see CHUNK above)
    xo, po, fo = sim.positions(), sim.momenta(), sim.forces()
    Uo = sim.energies()
    x_host.copy_(torch.from_numpy(xo)); p_host.copy_(torch.from_numpy(po)); f_host.copy_(torch.from_numpy(fo))
    xn, pn, fn = x_host.numpy(), p_host.numpy(), f_host.numpy()
    # device -> host results land in pinned buffers of their own (then become the next step's inputs)
    xo_h, po_h, fo_h = (torch.empty_like(x_host).pin_memory() for _ in range(3))
    xon, pon, fon = xo_h.numpy(), po_h.numpy(), fo_h.numpy()
    step_no = sim.estimators()["step"]
    e2e_steps = max(3, min(args.steps, 10))
    barrier()
    t0 = time.perf_counter()
    for q in range(e2e_steps):
        pk.pimd_restore(sim.ctx, xn, pn, fn, Uo, step_no + q)          # H2D: x, p, f (+U)
        sim.step(1)
        sim.positions(out=xon); sim.momenta(out=pon); sim.forces(out=fon)   # D2H
        Uo = sim.energies()
        est = sim.estimators()
        xn, xon = xon, xn; pn, pon = pon, pn; fn, fon = fon, fn            # results are the next step's inputs
    barrier()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    e2e_s = max_over_ranks(e2e_s, world, "cuda")
    h2d = 3 * P * N * 24 + P * 8
    d2h = 3 * P * N * 24 + P * 8 + 32

    out = None
    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            v, s_step, _, _ = _oracle_sample(args.config, 2, 1, 1)
            cpu = {"value": v, "unit": METRIC, "cores": _cores_used(), "kind": "oracle",
                   "sample": "configs[%d] box; 1 warm + 2 timed oracle steps with the force evaluation of 1 of %d beads "
                             "(%d bead-atoms per step); %.1f s/step" % (args.config, P, N, s_step)}
        out = {
            "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f16-split (3-pass hi/lo, f32 accumulate) network ~ f32 / f64 geometry+integrator", "data": "synthetic",
            "config": {"workload": cfg["name"] + ("+compressed_embedding" if args.compressed else ""), "atoms": N, "beads": P, "bead_atoms": P * N, "neighbour_rows": rows,
                       "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "ensemble": ("NpT %g bar, BZP barostat tau_p %g ps" % (cfg["p_ext_bar"], cfg["tau_p"])) if "p_ext_bar" in cfg else "NVT",
                       "l2": "no flush: per-step working set (neighbour rows %.0f MB, T and dT %.0f MB, fitting activations ~%.0f MB)%s" % (
                           rows * 32 / 1e6, 2 * P * N * 1600 / 1e6, P * N * 7740 / 1e6,
                           " exceeds the 126 MB L2" if rows * 32 + P * N * 3200 > 126e6 else " -- fits the 126 MB L2: small-case config, not a bench line")},
            "roofline": roofline, "kernels": kernels, "sustained": sustained, "compressed": compressed,
            "integrator_hbm": integ, "cpu_baseline": cpu,
            "e2e": {"value": world * P * N / e2e_s, "unit": METRIC, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_s * 1e3, "call": "pimd_restore(host x,p,f,U) + pimd_step(1) + pimd_get_{positions,momenta,forces,energies,estimators}"},
            "gpu_launches": int(launches), "clocks": clocks, "peaks": peaks,
            "paper_context": "fix pimd/langevin, 512 H2O x 32 beads: 2.56 M bead-atom-steps/s on 4xA100 (PAPER.md:L252, compressed DP model) -- context, not the target",
        }
        print(json.dumps(out))
    sim.close()
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


def integrator_leg(pk, peaks, n_atoms=1 << 20, P=32):
    """The fused integrator alone at a size that is HBM-bound: 2^20 atoms x 32 beads, harmonic
    model, 40 B per bead-atom-dim per launch -> 4.03 GB; the working set exceeds L2 so no flush is needed.
    Timed twice: with the PILE-L thermostat (the path of the benchmark) and at gamma = 0 (NVE: the same kernel
    without the O-step normals), which separates the memory system from the random-number arithmetic."""
    import torch
    rng = np.random.default_rng(0)
    types = np.zeros(n_atoms, np.int32)
    x = torch.from_numpy(rng.standard_normal((P, n_atoms, 3)) * 0.1).cuda()
    p = torch.from_numpy(rng.standard_normal((P, n_atoms, 3))).cuda()
    nbytes = 40.0 * 3 * n_atoms * P
    ms = {}
    for name, gamma in (("pile_l", 1.0), ("nve", 0.0)):
        sim = pk.PIMD(types, [1.008], [100.0] * 3, P, 300.0, 0.25e-3, gamma, seed=5)
        sim.set_model_harmonic(1.0)
        sim.set_state(x, p)
        ms[name] = pk.pimd_time_kernel(sim.ctx, 0, 10)
        if name == "pile_l":
            ms["per_mode_keying"] = pk.pimd_time_kernel(sim.ctx, 1, 10)      # DESIGN R-10's A/B partner (timing only)
        sim.close()
    del x, p
    torch.cuda.empty_cache()
    gbs = nbytes / (ms["pile_l"] * 1e-3) / 1e9
    gbs_nve = nbytes / (ms["nve"] * 1e-3) / 1e9
    return {"kernel": "integrator_kernel<32>", "bound": "hbm", "achieved": gbs, "peak": peaks["hbm"], "unit": "GB/s",
            "frac": gbs / peaks["hbm"], "ms": ms["pile_l"], "atoms": n_atoms, "beads": P, "bytes": nbytes,
            "nve": {"achieved": gbs_nve, "frac": gbs_nve / peaks["hbm"], "ms": ms["nve"]},
            "r10_ab": {"pair_keying_ms": ms["pile_l"], "per_mode_keying_ms": ms["per_mode_keying"],
                       "per_mode_frac": nbytes / (ms["per_mode_keying"] * 1e-3) / 1e9 / peaks["hbm"],
                       "note": "same launch with one Philox draw per mode (counter word 3 = 4k+alpha, sine branch "
                               "discarded: SURVEY C-7's first proposal) instead of one per mode pair (DESIGN R-10)"},
            "note": "stand-alone: closing B + estimators + B A O A + transforms; 'nve' = same launch at gamma = 0 "
                    "(no O-step normals): the gap is Philox + Box-Muller FP64 arithmetic, not memory"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json configs (default: the headline)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-integrator-leg", action="store_true")
    ap.add_argument("--no-compressed-leg", action="store_true", help="skip the compressed-embedding leg (SURVEY 8(f) NEXT-3)")
    ap.add_argument("--compressed", action="store_true",
                    help="time the compressed-embedding model as the main line (config.workload says so)")
    ap.add_argument("--no-tf32-peak", action="store_true", help="skip the cuBLAS TF32 peak measurement (roofline denominator)")
    ap.add_argument("--sustain-s", type=float, default=3.0,
                    help="seconds of back-to-back steps for the sustained-rate leg (0 = skip)")
    ap.add_argument("--integrator-only", action="store_true",
                    help="only the stand-alone integrator leg (2^20 atoms x 32 beads, HBM-bound size); prints its JSON")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.integrator_only:
        import paper_2602_13553_b200 as pk
        pk.lib()
        print(json.dumps(integrator_leg(pk, _peaks())))
        return 0
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
