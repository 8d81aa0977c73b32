#!/usr/bin/env python
"""bench.py — headline benchmark of gcoreccd-b200 (BASELINE.json: "Coulomb pair interactions/s (G/s) vs FP32
peak; seconds per 131k-hole event").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

A "step" is one pass of the whole hot path (field + integrate/collect + compact = SURVEY §8(a) rows a1..a8)
over the 131,072-hole cloud of BASELINE.json:configs[2].  Prints ONE JSON line (rank 0).
  value      pair interactions/s over the K timed steps, state resident in HBM, CUDA events on the launching
             stream, L2 flushed between timed steps (the state is only 2 MB; the path is ALU bound)
  e2e        same metric through the C ABI with HOST buffers: load_carriers(pinned host) + step(1) +
             read_carriers(host) per step, copies inside the timed region
  roofline   field kernel: 20 FLOP x pairs / CUDA-event duration of that kernel, against the FP32 non-tensor
             peak 148 SM x 128 lanes x 2 x sm_max_mhz
  cpu_baseline  the FP64 oracle, as it stands, on this box's host cores on a bounded sample of the same workload
N > 1: replicas only (BASELINE.json north_star: one GPU per event, no sharding): every rank runs its own
event; value = all ranks' pairs / max-over-ranks device time.
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

import numpy as np  # noqa: E402

METRIC = "coulomb_pair_interactions_per_s"
UNIT = "G pairs/s"
WORKLOAD_CFG = 2
FLOP_PER_PAIR = 20.0          # GPU Gems 3 ch. 31 convention (ref [10])
SM_COUNT, LANES = 148, 128


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """`nvidia-smi -lms 50` running beside the bench (B200_PROFILING.md clocks line); only the samples taken
    between mark_start() and mark_end() (the timed region, under load) are summarised."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.t0, self.t1, self.proc = index, [], None, None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"], stdout=subprocess.PIPE, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [t.strip() for t in line.split(",")]))

    def mark_start(self):
        self.t0 = time.perf_counter()

    def mark_end(self):
        self.t1 = time.perf_counter()

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        inside = [r for t, r in self.rows if self.t0 is not None and self.t0 <= t <= (self.t1 or t) + 0.06]
        sm, mx, reasons = [], 0.0, set()
        for r in inside:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm)}


# ----------------------------------------------------------------------------------------------- oracle legs
def oracle_sample(xyz, P, seconds_target, rng):
    """Time the oracle's eq. 6 double loop on m sampled targets x all sources; m sized for ~seconds_target."""
    from oracle import goracle as g
    n = len(xyz)
    Kp = g.coulomb_constant(P["eps_si"])
    x64 = xyz.astype(np.float64)
    m = 256
    t0 = time.perf_counter()
    g.coulomb_field(x64, eps_um=P["softening_um"], Kp=Kp, targets=np.arange(m, dtype=np.uint64))
    dt = time.perf_counter() - t0
    rate = m * n / dt
    m = int(max(256, seconds_target * rate / n))                     # may exceed n: targets are then revisited
    tg = np.sort(rng.integers(0, n, size=m)).astype(np.uint64)
    t0 = time.perf_counter()
    g.coulomb_field(x64, eps_um=P["softening_um"], Kp=Kp, targets=tg)
    dt = time.perf_counter() - t0
    return m * n / dt / 1e9, m, dt, g.num_threads()


def image_sigma(img, P):
    """Standard deviations (um) of the collected image along x and y, from pixel centres."""
    im = np.asarray(img, dtype=np.float64)
    ny, nx = im.shape
    xs = P["img_x0_um"] + (np.arange(nx) + 0.5) * P["pixel_pitch_um"]
    ys = P["img_y0_um"] + (np.arange(ny) + 0.5) * P["pixel_pitch_um"]
    tot = im.sum()
    mx, my = (im.sum(axis=0) * xs).sum() / tot, (im.sum(axis=1) * ys).sum() / tot
    return (np.sqrt((im.sum(axis=0) * (xs - mx) ** 2).sum() / tot), np.sqrt((im.sum(axis=1) * (ys - my) ** 2).sum() / tot))


def run_reference(args):
    """--impl reference: the FP64 oracle as it stands, on the host cores, same metric/unit/config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import goracle as g
    import workloads
    g.build()
    w = workloads.make(WORKLOAD_CFG)
    P, xyz = w["params"], w["xyz"]
    rng = np.random.default_rng(0)
    per_step_s = 3.0
    for _ in range(max(args.warmup, 0)):
        oracle_sample(xyz, P, 0.5, rng)
    pairs, secs, m_used = 0.0, 0.0, 0
    for _ in range(args.steps):
        gps, m, dt, cores = oracle_sample(xyz, P, per_step_s, rng)
        pairs += m * len(xyz); secs += dt; m_used = m
    value = pairs / secs / 1e9
    sample = "eq. 6 double loop (FP64) at %d sampled targets x all %d sources per step" % (m_used, len(xyz))
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": w["name"], "n_holes": len(xyz), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    import workloads
    from paper_2203_11043_b200 import binding, replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks, peak_src = measured_peaks()

    w = workloads.make(WORKLOAD_CFG, seed=replicas.rank_seed(workloads.SEED, rank))   # replicas: one event per rank
    P, xyz = w["params"], w["xyz"]
    n = len(xyz)
    stream = torch.cuda.Stream()                                       # the handle, the flush and the events share it
    torch.cuda.set_stream(stream)
    sim = binding.from_workload(w, stream=stream)
    sim.load_carriers(xyz)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(args.warmup):
        sim.step(1)
    barrier()
    l0 = sim.kernel_launches()
    p0 = sim.state()["pair_interactions"]
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    sampler.mark_start()
    for k in range(args.steps):
        flush.fill_(k & 0xff)                                          # L2 flush between timed iterations (untimed)
        ev[k][0].record()
        sim.step(1)
        ev[k][1].record()
    barrier()
    sampler.mark_end()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    clocks = sampler.stop() if rank == 0 else None
    launches = sim.kernel_launches() - l0
    st = sim.state()
    pairs = st["pair_interactions"] - p0
    ms_max, pairs_all = replicas.aggregate(ms, pairs, device="cuda")     # max over ranks of the device time, summed work
    value = pairs_all / (ms_max * 1e-3) / 1e9

    # ---- roofline of the dominant kernel (field), CUDA events inside the library on its launching stream
    prof = [sim.profile_step() for _ in range(max(3, min(args.steps, 10)))]
    n_act = sim.state()["n_active"]
    field_ms = float(np.mean([p["field"] for p in prof]))
    adv_ms = float(np.mean([p["advance"] for p in prof]))
    peak_tf = SM_COUNT * LANES * 2.0 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
    ach_tf = FLOP_PER_PAIR * float(n_act) ** 2 / (field_ms * 1e-3) / 1e12
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "field_traffic.json")) as f:
            traffic = json.load(f).get("dram_bytes_per_launch")
    except Exception:
        pass
    roofline = {"bound": "alu", "kernel": "k_field", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": ach_tf / peak_tf, "traffic": traffic, "peak_source": "148 SM x 128 FP32 lanes x 2 x sm_max_mhz (%s)" % peak_src,
                "flop_per_pair": FLOP_PER_PAIR, "field_ms": field_ms, "n_active": n_act,
                "other_kernels": {"advance_ms": adv_ms}}

    # ---- e2e through the C ABI with host buffers (copies inside the timed region)
    host_in = torch.from_numpy(xyz).pin_memory()
    host_out = torch.empty((n, 3), dtype=torch.float32).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    barrier()
    t0 = time.perf_counter()
    e2e_pairs = 0
    for _ in range(e2e_steps):
        sim.reset()
        sim.load_carriers_ptr(host_in.data_ptr(), n)
        sim.step(1)
        got = sim.read_carriers_into(host_out.data_ptr(), n)
        e2e_pairs += n * n
        assert got <= n
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_ms, e2e_pairs_all = replicas.aggregate(e2e_s * 1e3, e2e_pairs, device="cuda")
    e2e_value = e2e_pairs_all / (e2e_ms * 1e-3) / 1e9

    # ---- seconds per 131k-hole event (second half of BASELINE.json's metric): load -> full collection
    event = None
    if not args.no_event:
        runs = []
        for _ in range(3):                                  # best of 3 plus median
            sim.reset()
            barrier()
            t0 = time.perf_counter()
            sim.load_carriers_ptr(host_in.data_ptr(), n)
            done, left, rc = sim.run_to_collection(10 ** 7)
            img, over = sim.read_image()
            torch.cuda.synchronize()
            runs.append(time.perf_counter() - t0)
            st2 = sim.state()
            assert left == 0 and int(img.sum()) + over == n, "hole count not conserved"
        ev_s = min(runs)
        event = {"seconds": ev_s, "seconds_median": float(np.median(runs)), "runs": 3, "steps": done,
                 "pair_interactions": st2["pair_interactions"],
                 "avg_G_pairs_per_s": st2["pair_interactions"] / ev_s / 1e9, "holes": n, "collected_in_window": int(img.sum())}

    # ---- far-field VARIANT (reported separately, never part of `value`): same event, treecode
    farfield = None
    if not args.no_event and rank == 0 and event is not None:
        theta = 0.5
        sim.reset()
        sim.set_farfield(theta)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        sim.load_carriers_ptr(host_in.data_ptr(), n)
        done_f, left_f, rc = sim.run_to_collection(10 ** 7)
        img_f, over_f = sim.read_image()
        torch.cuda.synchronize()
        ff_s = time.perf_counter() - t0
        stf, ffs = sim.state(), sim.farfield_stats()
        assert left_f == 0 and int(img_f.sum()) + over_f == n, "hole count not conserved (far-field)"
        mom = lambda im: [float(v) for v in image_sigma(im, P)]
        farfield = {"theta": theta, "bound_B": ffs["bound_B"], "seconds": ff_s, "steps": done_f,
                    "interactions_evaluated": ffs["far_evals"] + ffs["near_evals"],
                    "fraction_of_all_pairs": (ffs["far_evals"] + ffs["near_evals"]) / float(stf["pair_interactions"]),
                    "speedup_vs_exact_event": event["seconds"] / ff_s,
                    "image_sigma_xy_um": mom(img_f), "exact_image_sigma_xy_um": mom(img),
                    "note": "approximate variant (treecode, monopole about the centre of charge); not the exact O(N^2) metric"}
        sim.set_farfield(-1.0)

    # ---- batched independent events (secondary numbers, not the headline): one CTA per event
    batched = None
    if not args.no_event and rank == 0:
        batched = []
        for sizes, what in (([2048] * 592, "592 X-ray events x 2,048 holes (7.5 keV-like clouds, sigma 0.5 um, depth U[10,665] um)"),
                            ([26] * 44400, "44,400 X-ray events x 26 holes (100 eV, PAPER.md:106)"),
                            ([4096] * 148, "148 events x 4,096 holes (few large events: one thread-block cluster per event)")):
            we = workloads.make_events(sizes)
            ne = len(we["xyz"])
            bs = binding.from_workload(we, max_carriers=ne, stream=stream)
            hin = torch.from_numpy(we["xyz"]).pin_memory()
            best = None
            for _ in range(2):
                bs.reset()
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                bs.load_events_ptr(hin.data_ptr(), we["offsets"])
                ev_left, ca_left, rc = bs.run_events()
                imgb, overb = bs.read_image()
                dt_s = time.perf_counter() - t0
                stb = bs.state()
                assert ca_left == 0 and int(imgb.sum()) + overb == ne, "hole count not conserved (batch)"
                if best is None or dt_s < best["seconds"]:
                    best = {"workload": what, "seconds": dt_s, "events_per_s": len(sizes) / dt_s,
                            "pair_interactions": stb["pair_interactions"],
                            "G_pairs_per_s": stb["pair_interactions"] / dt_s / 1e9,
                            "frac_of_fp32_peak": stb["pair_interactions"] * FLOP_PER_PAIR / dt_s / 1e12 / peak_tf,
                            "timing": "wall clock: load_events(pinned host) + run_events to full collection + read_image"}
            batched.append(best)
            bs.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- CPU baseline: the oracle as it stands on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import goracle as g
        g.build()
        gps, m, dt, cores = oracle_sample(xyz, P, 12.0, np.random.default_rng(0))
        cpu = {"value": gps, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "eq. 6 double loop (FP64) at %d sampled targets x all %d sources, %.1f s" % (m, n, dt)}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": w["name"], "n_holes": n, "parallelism": "replicas only (one event per GPU)",
                       "l2": "flushed between timed steps (256 MB write); state is 2 MB, path is ALU bound",
                       "dt_ns": P["dt_ns"], "softening_um": P["softening_um"]},
            "frac_of_fp32_peak": value * 1e9 * FLOP_PER_PAIR / 1e12 / (peak_tf * world),
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": n * 12, "d2h_bytes_per_step": n * 12,
                    "what": "reset + load_carriers(pinned host) + step(1) + read_carriers(host), wall clock"},
            "roofline": roofline, "cpu_baseline": cpu, "seconds_per_event": event, "farfield_variant": farfield,
            "batched_events": batched}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_sweep(args):
    """N sweep at fixed geometry (cfg-2 cloud), Coulomb on and off, 16 steps each through the graph path: the shape of
    the paper's Fig. 4 experiment.  One JSON line per size; not the headline number."""
    import torch
    import workloads
    from paper_2203_11043_b200 import binding
    peaks, _ = measured_peaks()
    peak_pairs = SM_COUNT * LANES * 2.0 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / FLOP_PER_PAIR
    sizes = [int(t) for t in args.sweep.split(",")]
    stream = torch.cuda.Stream()
    torch.cuda.set_stream(stream)
    for n in sizes:
        w = workloads.make(WORKLOAD_CFG, n=n)
        row = {"n": n}
        for name, flags in (("coulomb_on", 0), ("coulomb_off", binding.COULOMB_OFF)):
            sim = binding.from_workload(w, flags=flags, stream=stream)
            sim.load_carriers(w["xyz"])
            sim.step(8)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            best = 1e30
            for _ in range(3):
                e0.record(); sim.step(16); e1.record(); torch.cuda.synchronize()
                best = min(best, e0.elapsed_time(e1) / 16.0)
            row[name + "_ms_per_step"] = best
            if not flags:
                na = sim.state()["n_active"]
                row["G_pairs_per_s"] = na * float(na) / (best * 1e-3) / 1e9
                row["frac_of_fp32_peak"] = na * float(na) / (best * 1e-3) / peak_pairs
            sim.close()
        print(json.dumps(row), flush=True)
    return 0


def run_sharded(args):
    """--sharded CFG: ONE event's targets sharded over the ranks (not the headline, whose
    north_star fixes replicas).  Under torchrun: ShardedEvent over NCCL, strong scaling, device time max over ranks.
    On one GPU: --virtual-ranks G handles stepped sequentially; reports every rank's measured device time per step
    (shard_local + shard_commit, CUDA events) — the exchange over NVLink is NOT in that number."""
    import torch
    import torch.distributed as dist
    import workloads
    from paper_2203_11043_b200 import binding, replicas, sharded
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    w = workloads.make(int(args.sharded))
    xyz, n = w["xyz"], len(w["xyz"])
    stream = torch.cuda.Stream()
    torch.cuda.set_stream(stream)
    alloc = lambda nb: torch.empty(nb, dtype=torch.uint8, device="cuda")
    peaks, _ = measured_peaks()
    peak_pairs = SM_COUNT * LANES * 2.0 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / FLOP_PER_PAIR
    if world > 1 or args.exchange != "virtual":        # torchrun (any world size, also 1): the real multi-process path
        if not dist.is_initialized():
            if "RANK" not in os.environ:
                os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=os.environ.get("MASTER_PORT", "29511"), RANK="0", WORLD_SIZE="1")
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        if args.exchange == "symm":
            xf = lambda mb: sharded.SymmMemExchange(torch, "cuda", mb, world)
        else:
            xf = lambda mb: sharded.DistExchange(torch, "cuda", mb, world)
        ev = sharded.ShardedEvent(binding.from_workload(w, stream=stream), rank, world, xf, alloc)
        ev.load_carriers(xyz)
        if args.farfield >= 0:
            ev.e.set_farfield(args.farfield)
        ev.step(args.warmup)
        st0 = ev.refresh()
        dist.barrier(); torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); ev.step(args.steps); e1.record()
        dist.barrier(); torch.cuda.synchronize()
        tot = ev.totals(sharded.dist_reduce_sum(torch, "cuda"))
        ms, _ = replicas.aggregate(e0.elapsed_time(e1), 0.0, device="cuda")
        line = None
        if rank == 0:
            line = {"mode": "sharded", "n_gpus": world, "workload": w["name"], "n_holes": n, "steps": args.steps,
                    "ms_per_step": ms / args.steps, "n_active": tot["n_active"], "scaling": "strong",
                    "pair_interactions": tot["pair_interactions"],
                    "exchange": ("symmetric memory (peer loads in shard_commit)" if args.exchange == "symm" else
                                 "NCCL all_gather_into_tensor") + " of %d-byte messages" % ev.nbytes}
            print(json.dumps(line), flush=True)
        dist.destroy_process_group()
        return 0
    G = args.virtual_ranks
    es = [binding.from_workload(w, stream=stream) for _ in range(G)]
    vr = sharded.VirtualRanks(es, alloc)
    vr.load_carriers(xyz)
    if args.farfield >= 0:
        for e in es:
            e.set_farfield(args.farfield)
    vr.step(args.warmup)
    st = vr.refresh()
    na = st["n_active"]
    K = args.steps
    evs = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
            for _ in range(G)] for _ in range(K)]
    for k in range(K):                                    # VirtualRanks.step unrolled so each rank's kernels are bracketed
        msgs = vr.msgs[vr.k & 1]; vr.k += 1
        for g_, (e, m) in enumerate(zip(es, msgs)):
            evs[k][g_][0].record(); e.shard_local(m.data_ptr(), vr.nbytes); evs[k][g_][1].record()
        ptrs = [m.data_ptr() for m in msgs]
        for g_, e in enumerate(es):
            e.shard_commit(ptrs, vr.nbytes); evs[k][g_][2].record()
    torch.cuda.synchronize()
    local_ms = np.array([[evs[k][g_][0].elapsed_time(evs[k][g_][1]) for g_ in range(G)] for k in range(K)])
    commit_ms = np.array([[(evs[k][g_ - 1][2] if g_ else evs[k][G - 1][1]).elapsed_time(evs[k][g_][2]) for g_ in range(G)]
                          for k in range(K)])
    per_rank = (local_ms + commit_ms).mean(axis=0)
    st1 = vr.refresh()
    line = {"mode": "sharded-virtual", "farfield_theta": args.farfield if args.farfield >= 0 else None, "virtual_ranks": G, "workload": w["name"], "n_holes": n, "n_active_start": na,
            "n_active_end": st1["n_active"], "steps": K, "per_rank_ms_per_step": [float(v) for v in per_rank],
            "max_rank_ms_per_step": float(per_rank.max()), "sum_ranks_ms_per_step": float(per_rank.sum()),
            "commit_ms": float(commit_ms.mean()), "message_bytes": vr.nbytes,
            "frac_of_fp32_peak_per_rank": (float(na * float(na) / G / (per_rank.max() * 1e-3) / peak_pairs)
                                           if args.farfield < 0 else None),      # pairs evaluated only in the exact path
            "note": "each rank's kernels measured alone on one B200; the per-step all-gather of G messages over NVLink "
                    "is not included (one GPU available)"}
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-event", action="store_true", help="skip the seconds-per-event run")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", default="", help="comma-separated hole counts: per-step time vs N (not the headline)")
    ap.add_argument("--sharded", default="", help="config number: one event sharded over the ranks (not the headline)")
    ap.add_argument("--virtual-ranks", type=int, default=8, help="with --sharded on ONE GPU: ranks emulated sequentially")
    ap.add_argument("--farfield", type=float, default=-1.0, help="with --sharded: theta of the far-field variant (< 0: exact)")
    ap.add_argument("--exchange", default="virtual", choices=["virtual", "nccl", "symm"],
                    help="with --sharded: how the shard messages travel (virtual = one process, no exchange)")
    args = ap.parse_args()
    if args.sharded:
        return run_sharded(args)
    if args.sweep:
        return run_sweep(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
