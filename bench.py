#!/usr/bin/env python
"""bench.py — headline benchmark of gcoreccd-b200 (BASELINE.json: "Coulomb pair interactions/s (G/s) vs FP32
peak; seconds per 131k-hole event").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

A "step" is one pass of the whole hot path (k_field = a1, k_advance = a2..a8: update, collection, compaction; SURVEY
§8(a) rows a1..a8) over the 131,072-hole cloud of BASELINE.json:configs[2].  Prints ONE JSON line (rank 0).
  value      pair interactions/s over the K timed steps, state resident in HBM, CUDA events on the launching
             stream, L2 flushed between timed steps (the state is only 2 MB; the path is ALU bound)
  e2e        same metric through the C ABI with HOST buffers: load_carriers(pinned host) + step(1) +
             read_carriers(host) per step, copies inside the timed region
  roofline   field kernel: 20 FLOP x pairs / CUDA-event duration of that kernel, against the FP32 non-tensor
             peak 148 SM x 128 lanes x 2 x sm_max_mhz
  cpu_baseline  the FP64 oracle, as it stands, on this box's host cores on a bounded sample of the same workload
  per_config    configs 0-4 of BASELINE.json: per-step rate at step 0 and seconds per event (load -> full collection)
  n_sweep       per-step time against N = 2^10 .. 2^20 at the cfg-2 geometry, Coulomb on and off (Fig. 4)
  sharded_virtual  cfg3 sharded over 8 virtual ranks on this GPU (each rank's kernels timed alone)
N > 1: replicas only (BASELINE.json north_star: one GPU per event, no sharding): every rank runs its own
event; value = all ranks' pairs / max-over-ranks device time.  `python bench.py --gpus N` without torchrun spawns the
N ranks itself (one per device) and fails loudly if the box has fewer than N GPUs.  With N > 1 the line also carries a
`sharded` record: ONE cfg3 event's targets sharded over the N ranks (strong scaling, exchange included).
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

    def window(self, t0, t1):
        """Summary of the samples taken in [t0, t1] (a secondary leg's timed region)."""
        return self._summary([r for t, r in list(self.rows) if t0 <= t <= t1 + 0.06])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        return self._summary([r for t, r in self.rows if self.t0 is not None and self.t0 <= t <= (self.t1 or t) + 0.06])

    def _summary(self, inside):
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


def config_dict(w, n, P):
    """The same `config` for both arms (ours and --impl reference): the workload is what is compared."""
    return {"workload": w["name"], "n_holes": n, "parallelism": "replicas only (one event per GPU)",
            "l2": "flushed between timed steps (256 MB write); state is 2 MB, path is ALU bound",
            "dt_ns": P["dt_ns"], "softening_um": P["softening_um"]}


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
            "config": config_dict(w, len(xyz), P),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0



# ----------------------------------------------------------------------------------------------- secondary legs
def _peak_pairs(peaks):
    return SM_COUNT * LANES * 2.0 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / FLOP_PER_PAIR


def oracle_per_config(w, gpu_event):
    """the oracle's rate on this config (eq. 6 at sampled targets x all sources, ~2 s) and its
    seconds per event — run to completion for real on configs 0-1, extrapolated (the GPU run's sum of N_a^2 / the
    oracle's rate) on configs 2-4."""
    from oracle import goracle as g
    P, xyz = w["params"], w["xyz"]
    gps, m, dt, cores = oracle_sample(xyz, P, 2.0, np.random.default_rng(1))
    rec = {"G_pairs_per_s": gps, "cores": cores, "kind": "oracle (FP64)",
           "sample": "eq. 6 at %d sampled targets x all %d sources, %.1f s" % (m, len(xyz), dt)}
    if w["config"] <= 1:
        prm = g.make_params(T_K=P["T_K"], a1=P["a1"], a2=P["a2"], thickness_um=P["thickness_um"], z_well_um=P["z_well_um"],
                            pixel_pitch_um=P["pixel_pitch_um"], dt_ns=P["dt_ns"], softening_um=P["softening_um"],
                            eps_si=P["eps_si"], seed=P["seed"], img_nx=P["img_nx"], img_ny=P["img_ny"],
                            img_x0_um=P["img_x0_um"], img_y0_um=P["img_y0_um"], flags=g.FP32_STATE)
        sim = g.Sim(prm)
        t0 = time.perf_counter()
        sim.load(xyz)
        sim.run(10 ** 7)
        rec["seconds_per_event"] = time.perf_counter() - t0
        rec["seconds_per_event_kind"] = "measured (run to full collection, %d steps)" % sim.state()["step"]
        sim.close()
    else:
        rec["seconds_per_event"] = gpu_event["pair_interactions"] / (gps * 1e9)
        rec["seconds_per_event_kind"] = "extrapolated: the GPU run's sum of N_a^2 / the oracle's sampled rate"
    return rec


def leg_per_config(torch, binding, workloads, stream, peaks, sampler, configs=(0, 1, 2, 3, 4), reuse=None, with_oracle=False):
    """BASELINE.json configs 0-4 (north_star: "throughput on synthetic clouds and tracks ... as pair interactions/s, and
    as seconds per event"): per-step rate at step 0 (CUDA events around step(10) right after the load, best of 3) and
    seconds per event (wall clock: load_carriers from pinned host -> run_to_collection -> read_image; best of 3, cfg4
    once).  `reuse` = {cfg: event record} already measured by the caller (the headline's cfg2 event)."""
    peak = _peak_pairs(peaks)
    out = []
    for cfg in configs:
        w = workloads.make(cfg)
        xyz, n = w["xyz"], len(w["xyz"])
        sim = binding.from_workload(w, stream=stream)
        host_in = torch.from_numpy(xyz).pin_memory()
        t_leg0 = time.perf_counter()
        k_steps = 10
        best_ms, na0 = 1e30, 0
        for _ in range(3 if cfg < 4 else 2):
            sim.reset()
            sim.load_carriers_ptr(host_in.data_ptr(), n)
            st0 = sim.state()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); sim.step(k_steps); e1.record(); torch.cuda.synchronize()
            st1 = sim.state()
            ms = e0.elapsed_time(e1)
            if ms < best_ms:
                best_ms, pairs10, na0 = ms, st1["pair_interactions"] - st0["pair_interactions"], st0["n_active"]
        row = {"config": cfg, "workload": w["name"], "n_loaded": n, "n_active_at_step_0": na0,
               "ms_per_step_at_step_0": best_ms / k_steps,
               "G_pairs_per_s_at_step_0": pairs10 / (best_ms * 1e-3) / 1e9,
               "frac_of_fp32_peak_at_step_0": pairs10 / (best_ms * 1e-3) / peak}
        if reuse and cfg in reuse:
            row["event"] = reuse[cfg]
        else:
            runs = []
            for _ in range(3 if cfg < 4 else 1):
                sim.reset()
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                sim.load_carriers_ptr(host_in.data_ptr(), n)
                done, left, rc = sim.run_to_collection(10 ** 7)
                img, over = sim.read_image()
                torch.cuda.synchronize()
                runs.append(time.perf_counter() - t0)
                st2 = sim.state()
                assert left == 0 and int(img.sum()) + over == n, "hole count not conserved (cfg%d)" % cfg
            ev_s = min(runs)
            row["event"] = {"seconds": ev_s, "seconds_median": float(np.median(runs)), "runs": len(runs), "steps": done,
                            "pair_interactions": st2["pair_interactions"], "holes": n,
                            "avg_G_pairs_per_s": st2["pair_interactions"] / ev_s / 1e9,
                            "avg_frac_of_fp32_peak": st2["pair_interactions"] / ev_s / peak,
                            "collected_in_window": int(img.sum())}
        row["clocks"] = sampler.window(t_leg0, time.perf_counter())
        sim.close()
        if with_oracle:
            row["oracle"] = oracle_per_config(w, row["event"])
        out.append(row)
    return out


def leg_n_sweep(torch, binding, workloads, stream, peaks, sizes, persist_mode=1):
    """Per-step device time against N at the cfg-2 geometry, Coulomb on and off: the shape of the paper's Fig. 4
    experiment.  CUDA events around step(K) after a warm-up of 8 steps, best of 3."""
    peak = _peak_pairs(peaks)
    rows = []
    for n in sizes:
        w = workloads.make(WORKLOAD_CFG, n=n)
        row = {"n": n}
        for name, flags in (("coulomb_on", 0), ("coulomb_off", binding.COULOMB_OFF)):
            sim = binding.from_workload(w, flags=flags, stream=stream)
            if persist_mode != 1:
                sim.set_persistent(persist_mode)           # 0: two launches per step; 2: CTA-tile persistent kernels only
            sim.load_carriers(w["xyz"])
            # steps per timed call: a small population runs them all in ONE persistent launch, whose launch and exit
            # (~10 us) would otherwise be a visible share of 16 steps of 7-15 us; events run hundreds of steps per launch
            k = 64 if (not flags and n <= 16384) else 16 if (flags or n <= 131072) else 4
            sim.step(8 if n <= 131072 else 2)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            best = 1e30
            for _ in range(3 if n <= 262144 else 2):
                e0.record(); sim.step(k); e1.record(); torch.cuda.synchronize()
                best = min(best, e0.elapsed_time(e1) / k)
            row[name + "_us_per_step"] = best * 1e3
            if not flags:
                na = sim.state()["n_active"]
                row["G_pairs_per_s"] = na * float(na) / (best * 1e-3) / 1e9
                row["frac_of_fp32_peak"] = na * float(na) / (best * 1e-3) / peak
            sim.close()
        rows.append(row)
    return rows


def leg_sharded_virtual(torch, binding, workloads, sharded, stream, peaks, cfg, G, steps, warmup, farfield=-1.0):
    """ONE event's targets sharded over G virtual ranks on ONE GPU: the ranks' kernels run one
    after the other on one stream and are timed separately (shard_local + shard_commit, CUDA events); the per-step
    all-gather over NVLink is NOT in these numbers (one GPU available)."""
    w = workloads.make(int(cfg))
    xyz, n = w["xyz"], len(w["xyz"])
    alloc = lambda nb: torch.empty(nb, dtype=torch.uint8, device="cuda")
    es = [binding.from_workload(w, stream=stream) for _ in range(G)]
    vr = sharded.VirtualRanks(es, alloc)
    vr.load_carriers(xyz)
    if farfield >= 0:
        for e in es:
            e.set_farfield(farfield)
    vr.step(warmup)
    st = vr.refresh()
    na = st["n_active"]
    K = steps
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
    rec = {"mode": "sharded-virtual", "farfield_theta": farfield if farfield >= 0 else None, "virtual_ranks": G,
           "workload": w["name"], "n_holes": n, "n_active_start": na, "n_active_end": st1["n_active"], "steps": K,
           "per_rank_ms_per_step": [float(v) for v in per_rank],
           "max_rank_ms_per_step": float(per_rank.max()), "sum_ranks_ms_per_step": float(per_rank.sum()),
           "commit_ms": float(commit_ms.mean()), "message_bytes": vr.nbytes,
           "frac_of_fp32_peak_per_rank": (float(na * float(na) / G / (per_rank.max() * 1e-3) / _peak_pairs(peaks))
                                          if farfield < 0 else None),      # pairs evaluated only in the exact path
           "note": "each rank's kernels measured alone on one B200; the per-step all-gather of G messages over NVLink "
                   "is not included (one GPU available)"}
    for e in es:
        e.close()
    return rec


def leg_sharded_real(torch, dist, binding, workloads, sharded, replicas, stream, rank, world, cfg, steps, warmup, exchange):
    """ONE event sharded over the `world` ranks of this job (torchrun / --gpus N): strong scaling, device time of
    `steps` sharded steps, exchange (NCCL all-gather, or symmetric-memory peer loads) included, max over ranks."""
    w = workloads.make(int(cfg))
    alloc = lambda nb: torch.empty(nb, dtype=torch.uint8, device="cuda")
    if exchange == "symm":
        xf = lambda mb: sharded.SymmMemExchange(torch, "cuda", mb, world)
    else:
        xf = lambda mb: sharded.DistExchange(torch, "cuda", mb, world)
    ev = sharded.ShardedEvent(binding.from_workload(w, stream=stream), rank, world, xf, alloc)
    ev.load_carriers(w["xyz"])
    ev.step(warmup)
    st0 = ev.refresh()
    dist.barrier(); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); ev.step(steps); e1.record()
    dist.barrier(); torch.cuda.synchronize()
    tot = ev.totals(sharded.dist_reduce_sum(torch, "cuda"))
    ms, _ = replicas.aggregate(e0.elapsed_time(e1), 0.0, device="cuda")
    ev.e.close()
    return {"mode": "sharded", "n_gpus": world, "workload": w["name"], "n_holes": len(w["xyz"]), "steps": steps,
            "ms_per_step": ms / steps, "n_active_start": st0["n_active"], "n_active": tot["n_active"], "scaling": "strong",
            "pair_interactions": tot["pair_interactions"],
            "exchange": ("symmetric memory (peer loads in shard_commit)" if exchange == "symm" else
                         "NCCL all_gather_into_tensor") + " of %d-byte messages" % ev.nbytes}


# ----------------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    import workloads
    from paper_2203_11043_b200 import binding, replicas, sharded

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
    clocks = sampler.window(sampler.t0, sampler.t1) if rank == 0 else None
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
    traffic, traffic_src, adv_inst = None, None, None
    try:                                                               # NOT measured by this run: a stored ncu capture
        with open(os.path.join(ROOT, "profiles", "field_traffic.json")) as f:
            tj = json.load(f)
        traffic, adv_inst = tj.get("dram_bytes_per_launch"), tj.get("advance_warp_inst_per_warp")
        traffic_src = "static: profiles/field_traffic.json (%s)" % tj.get("source", "ncu capture")
    except Exception:
        pass
    # a2..a8 (k_advance): not bound by HBM (its bytes are L2-resident) and not by FP64 throughput (pipe 14 % busy) but by
    # the latency of a ~1,500-instruction dependent chain per carrier at 0.86 waves; the floor quoted is
    # the instruction-issue time of that stream: warps x instructions / (SMs x 4 schedulers x clock)
    clock_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    issue_floor_ms = (adv_inst * (n_act / 32.0) / (SM_COUNT * 4.0 * clock_hz) * 1e3) if adv_inst else None
    adv = {"kernel": "k_advance", "ms": adv_ms, "algorithmic_bytes_per_carrier": 32 + 12 * 16,
           "GBps_of_algorithmic_bytes": (32.0 + 12.0 * 16) * n_act / (adv_ms * 1e-3) / 1e9, "hbm_peak_GBps": peaks.get("hbm_gbs"),
           "frac_of_hbm_peak": (32.0 + 12.0 * 16) * n_act / (adv_ms * 1e-3) / 1e9 / float(peaks.get("hbm_gbs", 6650.0)),
           "bound": "latency of the per-carrier dependent chain (L2 round trips of the chunk partials + FP64 update), 0.86 waves",
           "warp_inst_per_warp": adv_inst, "issue_floor_ms": issue_floor_ms,
           "frac_of_issue_floor": (issue_floor_ms / adv_ms) if issue_floor_ms else None}
    roofline = {"bound": "alu", "kernel": "k_field", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": ach_tf / peak_tf, "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": "148 SM x 128 FP32 lanes x 2 x sm_max_mhz (%s)" % peak_src,
                "flop_per_pair": FLOP_PER_PAIR, "field_ms": field_ms, "n_active": n_act,
                "other_kernels": {"advance": adv}}

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

    def _line(sharded_rec, cpu, per_config, n_sweep, sharded_virtual):
        return {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": config_dict(w, n, P),
                "frac_of_fp32_peak": value * 1e9 * FLOP_PER_PAIR / 1e12 / (peak_tf * world),
                "clocks": clocks, "gpu_launches": launches,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": n * 12, "d2h_bytes_per_step": n * 12,
                        "what": "reset + load_carriers(pinned host) + step(1) + read_carriers(host), wall clock"},
                "roofline": roofline, "cpu_baseline": cpu, "seconds_per_event": event, "farfield_variant": farfield,
                "batched_events": batched, "per_config": per_config, "n_sweep": n_sweep, "sharded_virtual": sharded_virtual,
                "sharded": sharded_rec}

    # ---- ONE event sharded over the job's ranks (N > 1 only; strong scaling; not the headline, which is replicas)
    # This leg has never run on more than one GPU (the build's boxes have one): it must not be able to take the headline
    # with it.  A watchdog prints the line without it (rank 0) and ends the rank if the leg hangs; an exception on
    # any rank is caught and reported the same way.
    sharded_rec = None
    if world > 1 and not args.no_event:
        import threading

        def _bail():
            if rank == 0:
                print(json.dumps(_line({"error": "the sharded leg did not finish within 300 s"}, None, None, None, None)), flush=True)
            os._exit(0)
        wd = threading.Timer(300.0, _bail)
        wd.daemon = True
        wd.start()
        try:
            sharded_rec = leg_sharded_real(torch, dist, binding, workloads, sharded, replicas, stream, rank, world, 3,
                                           max(8, args.steps), args.warmup, "nccl")
        except Exception as e:                                # noqa: BLE001 - reported in the line, never fatal
            sharded_rec = {"error": repr(e)[:400]}
        wd.cancel()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- every config, the N sweep, 8 virtual ranks (rank 0, N = 1; each leg clock-sampled like the headline)
    per_config = n_sweep = sharded_virtual = None
    if world == 1 and not args.no_event and not args.quick:
        per_config = leg_per_config(torch, binding, workloads, stream, peaks, sampler,
                                    reuse={2: dict(event, avg_frac_of_fp32_peak=event["avg_G_pairs_per_s"] * 1e9 / _peak_pairs(peaks))},
                                    with_oracle=not args.no_cpu_baseline)
        t0 = time.perf_counter()
        n_sweep = {"rows": leg_n_sweep(torch, binding, workloads, stream, peaks, [2 ** k for k in range(10, 21)]),
                   "what": "cfg-2 geometry, us per step through gcoreccd_step (CUDA events, best of 3), Coulomb on / off"}
        n_sweep["clocks"] = sampler.window(t0, time.perf_counter())
        t0 = time.perf_counter()
        sharded_virtual = leg_sharded_virtual(torch, binding, workloads, sharded, stream, peaks, 3, 8, 8, 3)
        sharded_virtual["clocks"] = sampler.window(t0, time.perf_counter())
    sampler.stop()

    # ---- CPU baseline: the oracle as it stands on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import goracle as g
        g.build()
        gps, m, dt, cores = oracle_sample(xyz, P, 12.0, np.random.default_rng(0))
        cpu = {"value": gps, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "eq. 6 double loop (FP64) at %d sampled targets x all %d sources, %.1f s" % (m, n, dt)}

    line = _line(sharded_rec, cpu, per_config, n_sweep, sharded_virtual)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_sweep(args):
    """--sweep N,...: the n_sweep leg alone, one JSON line per size (not the headline number)."""
    import torch
    import workloads
    from paper_2203_11043_b200 import binding
    peaks, _ = measured_peaks()
    stream = torch.cuda.Stream()
    torch.cuda.set_stream(stream)
    for row in leg_n_sweep(torch, binding, workloads, stream, peaks, [int(t) for t in args.sweep.split(",")],
                           persist_mode=args.persist_mode):
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
    stream = torch.cuda.Stream()
    torch.cuda.set_stream(stream)
    peaks, _ = measured_peaks()
    if world > 1 or args.exchange != "virtual":        # torchrun (any world size, also 1): the real multi-process path
        if not dist.is_initialized():
            if "RANK" not in os.environ:
                os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=os.environ.get("MASTER_PORT", "29511"), RANK="0", WORLD_SIZE="1")
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        rec = leg_sharded_real(torch, dist, binding, workloads, sharded, replicas, stream, rank, world, int(args.sharded),
                               args.steps, args.warmup, args.exchange)
        if rank == 0:
            print(json.dumps(rec), flush=True)
        dist.destroy_process_group()
        return 0
    rec = leg_sharded_virtual(torch, binding, workloads, sharded, stream, peaks, int(args.sharded), args.virtual_ranks,
                              args.steps, args.warmup, args.farfield)
    print(json.dumps(rec), flush=True)
    return 0


def run_microbench(args):
    """--microbench: instruction-throughput probes behind DESIGN.md 6.1 / 6.8 (one SM; cycles per warp-instruction per
    SM sub-partition; 2.0 = a packed FP32x2 instruction at full lane rate).  One JSON line."""
    from paper_2203_11043_b200 import binding
    rows = []
    for kind, name in enumerate(binding.MICRO_KINDS):
        rows.append({"kind": name, **{"warps_%d" % w: round(binding.microbench(kind, 4096, w), 3) for w in (1, 2, 4)}})
    print(json.dumps({"microbench": rows, "unit": "cycles per warp-instruction per SM sub-partition"}), flush=True)
    return 0


def _spawned(local_rank, args, port):
    os.environ.update(RANK=str(local_rank), LOCAL_RANK=str(local_rank), WORLD_SIZE=str(args.gpus),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.exit(dispatch(args))


def spawn_ranks(args):
    """`python bench.py --gpus N` without torchrun: one process per GPU of this node, same code path as under torchrun."""
    import socket
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        sys.stderr.write("bench.py: --gpus %d asked for but this box has %d CUDA device(s); refusing to run fewer ranks "
                         "than asked (launch on a node with %d GPUs, or pass --gpus %d)\n" % (args.gpus, have, args.gpus, max(have, 1)))
        return 2
    with socket.socket() as s_:
        s_.bind(("127.0.0.1", 0))
        port = s_.getsockname()[1]
    import torch.multiprocessing as mp
    mp.spawn(_spawned, args=(args, port), nprocs=args.gpus, join=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-event", action="store_true", help="skip the seconds-per-event run")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--microbench", action="store_true", help="instruction-throughput probes (DESIGN.md 6.1 / 6.8)")
    ap.add_argument("--quick", action="store_true", help="skip the per_config / n_sweep / sharded_virtual legs")
    ap.add_argument("--persist-mode", type=int, default=1, choices=[0, 1, 2],
                    help="with --sweep: 0 two launches per step, 2 persistent CTA-tile kernels only, 1 default")
    ap.add_argument("--sweep", default="", help="comma-separated hole counts: per-step time vs N (not the headline)")
    ap.add_argument("--sharded", default="", help="config number: one event sharded over the ranks (not the headline)")
    ap.add_argument("--virtual-ranks", type=int, default=8, help="with --sharded on ONE GPU: ranks emulated sequentially")
    ap.add_argument("--farfield", type=float, default=-1.0, help="with --sharded: theta of the far-field variant (< 0: exact)")
    ap.add_argument("--exchange", default="virtual", choices=["virtual", "nccl", "symm"],
                    help="with --sharded: how the shard messages travel (virtual = one process, no exchange)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference" and not args.sweep:
        return spawn_ranks(args)
    if "WORLD_SIZE" in os.environ and int(os.environ["WORLD_SIZE"]) != args.gpus and not args.sharded:
        sys.stderr.write("bench.py: --gpus %d but WORLD_SIZE=%s\n" % (args.gpus, os.environ["WORLD_SIZE"]))
        return 2
    return dispatch(args)


def dispatch(args):
    if args.microbench:
        return run_microbench(args)
    if args.sharded:
        return run_sharded(args)
    if args.sweep:
        return run_sweep(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
