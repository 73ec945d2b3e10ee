#!/usr/bin/env python
"""bench.py -- ps per spin-flip attempt (paper Eq. 2) on BASELINE.json's
headline workload (config 4: L=16, 2048 realizations x 24 temperatures, PT every sweep),
through the C ABI of libea_b200.so.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--sweeps-per-step 5000]
                  (N > 1 without a launcher: re-executes itself under torch.distributed.run)
  python bench.py --impl reference ...      # the CPU oracle, as it stands, on the host cores
  python bench.py --field 1                 # the same workload with h = 1 (generic kernel)
  python bench.py --measure-every 10        # two-copy overlap/energy moments every 10 sweeps
  python bench.py --swap-mode move                         # swaps that move the lattices
  python bench.py --layout replica --sweeps-per-step 200   # the paper's own coding (bits = temperature
                                            # replicas of one realization, one random number per replica)

A *step* = `sweeps_per_step` full checkerboard sweeps, each followed by a PT round (config's
swap_interval), of the whole workload: every row of SURVEY.md section 8(a) on the hot path.
One JSON line on stdout (rank 0).  Details: DESIGN.md section 8.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from ea_inputs import CONFIGS, betas_for  # noqa: E402

METRIC = "ps per spin-flip attempt"
UNIT = "ps/attempt"
# ALU-pipe (LOP3/IADD/SHF/ISETP class) lane-operations the method needs per word update
# (32 attempts), derived in DESIGN.md section 8: 30 on every update + 15.5 on parity-1 updates
# (energy).  Philox's multiplies and the table addressing run on the FMA pipe and are not
# counted; the kernels execute ~47 ALU instructions per update (profiles/).
ALU_OPS_PER_WORD_UPDATE = 38.0
PAPER_PS = 33.5   # GTX 580, PT every 10 sweeps: context, another workload
# ncu --set full summaries of the dominant kernel, committed under profiles/ (tracked text): DRAM
# bytes per launch and the ALU pipe's busy share are READ from them at run time, and only for the
# workload the capture was taken on (default shape of that config, no field, no measurement
# series); any other workload reports traffic = null.  tests/test_bench_host.py ties the parser to
# the files.
NCU_PROFILES = {4: ("r02_ncu_resident_cfg4.txt", "k_resident"), 5: ("r02_ncu_stream_cfg5.txt", "k_stream")}


def ncu_profile_numbers(config):
    """{'dram_bytes': read + write per launch, 'alu_pipe_max_pct': ..., 'file': ...} or None."""
    ent = NCU_PROFILES.get(config)
    if not ent:
        return None
    path = os.path.join(ROOT, "profiles", ent[0])
    if not os.path.exists(path):
        return None
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    out = {"file": "profiles/" + ent[0], "dram_bytes": 0.0, "alu_pipe_max_pct": None}
    seen = 0
    for line in open(path):
        f = line.split()
        if len(f) >= 3 and f[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum") and f[1] in unit:
            out["dram_bytes"] += float(f[2]) * unit[f[1]]; seen += 1
        if len(f) >= 3 and f[0] == "sm__inst_executed_pipe_alu.max.pct_of_peak_sustained_active":
            out["alu_pipe_max_pct"] = float(f[-1])
    return out if seen == 2 else None


# ---- golden digests (tests/golden, written by the CPU oracle alone): the timed trajectory is
# checked against them ("every repeat ... must end in the same digest")
def golden_checkpoints(config):
    """{word: {sweeps: digest}} of the oracle digests stored for `config`."""
    import glob
    out = {}
    for f in glob.glob(os.path.join(ROOT, "tests", "golden", f"digests_cfg{config}_w*.json")):
        g = json.load(open(f))
        out[int(g["word"])] = {int(c): v["digest"] for c, v in g["checkpoints"].items()}
    return out


def check_digest(sim, cfg, config, done):
    """Sweep on (untimed) from `done` to the first stored checkpoint >= done and compare the digest
    of every word that has one there.  Returns a dict for the JSON line; 'ok' is None when no
    checkpoint lies ahead."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from util_pack import word_digest
    gold = golden_checkpoints(config)
    ahead = sorted({c for w in gold.values() for c in w if c >= done})
    if not ahead:
        return {"ok": None, "why": "no oracle digest at or after sweep %d" % done}
    cp = ahead[0]
    if cp > done:
        sim.sweep(cp - done, cfg.swap_interval)
    st = sim.get_state()
    words, ok = [], True
    for w, cps in sorted(gold.items()):
        if cp not in cps or w >= cfg.W:
            continue
        Rw = min(32, cfg.R - 32 * w)
        mask = np.uint32((1 << Rw) - 1) if Rw < 32 else np.uint32(0xFFFFFFFF)
        d = word_digest(st["spin_words"][:, w] & mask, st["temp_of_slot"][32 * w:32 * w + Rw],
                        st["energy_by_slot"][32 * w:32 * w + Rw])
        words.append(w)
        ok = ok and d == cps[cp]
    return {"ok": bool(ok) if words else None, "sweep": cp, "timed_sweeps": done, "words": words,
            "source": "tests/golden/digests_cfg%d_w*.json (CPU oracle)" % config}


def _clock_sampler(stop, out):
    q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    dev = os.environ.get("LOCAL_RANK", "0")
    while not stop.is_set():
        try:
            r = subprocess.run(["nvidia-smi", "-i", dev, f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                               capture_output=True, text=True, timeout=5)
            if r.returncode == 0 and r.stdout.strip():
                out.append([x.strip() for x in r.stdout.strip().split(",")])
        except Exception:
            pass
        stop.wait(0.1)


def _clock_summary(samples):
    sm, mx, reasons = [], [], set()
    names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    for s in samples:
        try:
            sm.append(float(s[1])); mx.append(float(s[2]))
        except Exception:
            continue
        for name, v in zip(names, s[5:9]):
            if v.lower().startswith("active"):
                reasons.add(name)
    if not sm:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
    return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
            "samples": len(sm)}


# ------------------------------------------------------------------ CPU oracle legs
def _oracle_worker(args):
    L, nT, betas, seed, r0, sweeps, swap, field = args
    from oracle import Oracle
    o = Oracle(L, nT, 32, betas, seed, r0=r0)
    if field:
        o.set_field(field)
    t = time.perf_counter()
    o.sweep(sweeps, swap)
    return time.perf_counter() - t


def oracle_sample(cfg, words, sweeps, procs, field=0):
    """Time the oracle, as it stands, on `words` realization words of cfg (one word = 32
    realizations, all temperatures) for `sweeps` sweeps, `procs` processes (one word each at a
    time).  Returns (ps per attempt over the wall time, wall seconds)."""
    import multiprocessing as mp
    from oracle import build_oracle
    build_oracle()
    betas = betas_for(cfg)
    jobs = [(cfg.L, cfg.n_temps, betas, cfg.seed, 32 * w, sweeps, cfg.swap_interval, field) for w in range(words)]
    t = time.perf_counter()
    if procs == 1:
        for j in jobs:
            _oracle_worker(j)
    else:
        with mp.get_context("fork").Pool(procs) as pool:
            pool.map(_oracle_worker, jobs, chunksize=1)
    wall = time.perf_counter() - t
    attempts = words * 32 * cfg.n_temps * cfg.N * sweeps
    return wall * 1e12 / attempts, wall


def run_reference(a, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = len(os.sched_getaffinity(0)) if not a.ref_cores else a.ref_cores
    words = min(cores, cfg.W)
    sweeps = max(1, int(1.5e8 / (32 * cfg.n_temps * cfg.N)))      # ~4 s of one core per word
    for _ in range(max(a.warmup, 1)):           # at least once: builds the oracle, starts the pool
        oracle_sample(cfg, words, 1, words, a.field)
    vals, walls = [], []
    for _ in range(a.steps):
        v, wsec = oracle_sample(cfg, words, sweeps, words, a.field)
        vals.append(v); walls.append(wsec)
    value = float(np.mean(vals))
    sample = f"{words} of {cfg.W} words (32 realizations x {cfg.n_temps} temperatures each) x {sweeps} sweeps per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": a.gpus,
        "steps": a.steps, "warmup": a.warmup, "ms_per_step": float(np.mean(walls)) * 1e3,
        "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "int8 spins / u32 draws",
        "data": "synthetic", "config": {"workload": cfg.name, "L": cfg.L, "n_temps": cfg.n_temps,
                                        "realizations": cfg.R, "swap_interval": cfg.swap_interval,
                                        "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": words, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ------------------------------------------------------------------ multi-GPU plumbing
def shard_first_realization(rank, realizations_per_rank):
    """Weak scaling by realization word: rank r owns global realizations [r*R, (r+1)*R), R a
    multiple of 32 per rank except possibly the last word (counters are keyed by the GLOBAL word
    index, so the union of the ranks equals one big single-process run)."""
    words = (realizations_per_rank + 31) // 32
    return rank * words * 32


def max_over_ranks(ms, world, device="cuda"):
    """Timing of a multi-rank run = the slowest rank (all-reduce MAX)."""
    if world == 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# ------------------------------------------------------------------ CUDA arm
KERNEL_NAMES = {1: "generic", 2: "resident", 3: "tiled", 4: "stream"}


def alu_ops_per_update(cfg, sps):
    """30 on every update + 7.75 for the energy pass, which only runs on sweeps followed by a swap
    round (and the last sweep of a call): 38 for the configs' PT every sweep."""
    e_frac = (1.0 / cfg.swap_interval) if cfg.swap_interval > 0 else 1.0 / sps
    return 30.0 + (ALU_OPS_PER_WORD_UPDATE - 30.0) * e_frac


def hbm_view(cfg, sps, step_s):
    """Streaming kernel: algorithmic bytes = per half-sweep and item, tile read (own parity + other
    parity with halo) + own parity written back; the state fits L2, so this is L2 traffic and the
    HBM figure is context, not the bound."""
    zs = 512 // ((cfg.L // 8) * cfg.L)
    tile = 512 * 16 + (zs + 2) * (cfg.L // 8) * cfg.L * 16 + 512 * 16
    bytes_step = 2.0 * tile * cfg.n_temps * cfg.W * (cfg.L // zs) * sps
    peaks = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm = json.load(open(peaks))["hbm_gbs"] if os.path.exists(peaks) else 6650.0
    gbs = bytes_step / step_s / 1e9
    return {"algorithmic_GBps": gbs, "peak_GBps": hbm, "frac": gbs / hbm,
            "peak_source": "MEASURED_PEAKS.json" if os.path.exists(peaks) else "B200_PROFILING.md fallback",
            "note": "tile bytes streamed per sweep / time; served by L2 (state 35 MiB < 126 MB)"}


def time_steps(torch, sim, step, steps, flush_l2):
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for e0, e1 in ev:
        flush_l2()
        e0.record()
        step()
        e1.record()
    torch.cuda.synchronize()
    return [e0.elapsed_time(e1) for e0, e1 in ev]


def oracle_one_core(cfg):
    """The oracle on ONE host core on this config's shape: one word (or the config's R if smaller),
    about 1e8 attempts (~1 s)."""
    from oracle import Oracle, build_oracle
    build_oracle()
    R = min(32, cfg.R)
    sweeps = max(1, int(1.0e8 / (R * cfg.n_temps * cfg.N)))
    o = Oracle(cfg.L, cfg.n_temps, R, betas_for(cfg), cfg.seed)
    t = time.perf_counter()
    o.sweep(sweeps, cfg.swap_interval)
    return (time.perf_counter() - t) * 1e12 / (R * cfg.n_temps * cfg.N * sweeps)


def per_config_block(torch, EA, flush_l2, lop3_peak, skip):
    """ps per attempt on every BASELINE config, outside the headline's timed region:
    3 steps of 1000 sweeps each (config 1: 333, its full length) on a fresh handle after one warm-up step,
    and the trajectory checked against the oracle's digest at the next stored checkpoint."""
    out = {}
    for cid in (1, 2, 3, 4, 5):
        if cid == skip:
            continue
        cfg = CONFIGS[cid]
        sps = min(1000, cfg.sweeps // 3)
        warm = EA(cfg.L, cfg.n_temps, cfg.R, betas_for(cfg), cfg.seed)
        warm.sweep(sps, cfg.swap_interval)
        warm.synchronize()
        warm.destroy()
        sim = EA(cfg.L, cfg.n_temps, cfg.R, betas_for(cfg), cfg.seed)
        ms = time_steps(torch, sim, lambda: sim.sweep(sps, cfg.swap_interval), 3, flush_l2)
        step_s = float(np.mean(ms)) * 1e-3
        ops = alu_ops_per_update(cfg, sps) * cfg.n_temps * cfg.W * cfg.N * sps
        ent = {"workload": cfg.name, "kernel": KERNEL_NAMES.get(sim.get_kernel()), "sweeps_per_step": sps,
               "us_per_sweep": step_s * 1e6 / sps, "ps_per_attempt": step_s * 1e12 / (cfg.attempts_per_sweep * sps),
               "alu_frac": ops / step_s / lop3_peak, "digest": check_digest(sim, cfg, cid, 3 * sps)}
        if sim.get_kernel() == 4:
            ent["hbm_view"] = hbm_view(cfg, sps, step_s)
        ent["oracle_one_core_ps"] = oracle_one_core(cfg)
        out[str(cid)] = ent
        sim.destroy()
    return out


def run_cuda(a, cfg):
    import torch
    import torch.distributed as dist
    from paper_1311_5582_b200 import EA, measure_int_peak

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert a.gpus == world, f"--gpus {a.gpus} but WORLD_SIZE is {world}"
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    betas = betas_for(cfg)
    sps = a.sweeps_per_step
    me = a.measure_every
    # the golden digests describe the BASELINE config itself, as rank 0 simulates it
    replica = a.layout == "replica"
    moving = a.swap_mode == "move"
    plain = not (a.field or me or a.realizations is not None or a.swap_interval is not None or replica or moving)

    def make():
        # weak scaling: every rank owns cfg.R realizations; rank r simulates global words r*W..
        sim = EA(cfg.L, cfg.n_temps, cfg.R, betas, cfg.seed, first_realization=shard_first_realization(rank, cfg.R))
        if a.field:
            sim.set_field(a.field)
        if replica:
            from paper_1311_5582_b200 import EA_LAYOUT_REPLICA_BITS
            sim.set_layout(EA_LAYOUT_REPLICA_BITS)
        if moving:
            from paper_1311_5582_b200 import EA_SWAP_MOVE
            sim.set_swap_mode(EA_SWAP_MOVE)
        if me:
            # two copies of every disorder realization (words w and w + W/2), overlap and energy
            # moments accumulated on the device every `me` sweeps (ea_measure)
            assert cfg.R % 64 == 0 and sps % me == 0, "--measure-every needs R % 64 == 0 and sweeps-per-step % M == 0"
            sim.pair_couplings()
            sim.measure_begin([[w, w + cfg.W // 2] for w in range(cfg.W // 2)])
        return sim

    def stepper(sim):
        if me:
            return lambda: sim.measure(sps // me, me, cfg.swap_interval)
        return lambda: sim.sweep(sps, cfg.swap_interval)

    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def flush_l2():
        flush.add_(1)

    # ---- warm-up on a handle of its own, so that the timed handle starts from sweep 0 and its
    #      trajectory can be compared with the oracle's digests afterwards
    warm = make()
    wstep = stepper(warm)
    for _ in range(a.warmup):
        wstep()
    warm.synchronize()
    warm.destroy()
    sim = make()
    step = stepper(sim)
    kernel = sim.get_kernel()

    # ---- kernel-resident timing: state in HBM/SMEM, no host buffers
    barrier()
    samples, stop = [], threading.Event()
    th = threading.Thread(target=_clock_sampler, args=(stop, samples), daemon=True)
    th.start()
    launches0 = sim.launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(a.steps)]
    barrier()
    for e0, e1 in ev:
        flush_l2()
        e0.record()
        step()
        e1.record()
    barrier()
    stop.set(); th.join()
    launches = sim.launch_count() - launches0
    step_ms = [e0.elapsed_time(e1) for e0, e1 in ev]
    total_ms = max_over_ranks(float(sum(step_ms)), world)
    attempts_step = cfg.attempts_per_sweep * sps * world
    value = total_ms * 1e9 / (attempts_step * a.steps)            # ms -> ps

    # ---- the timed trajectory against the CPU oracle's digests (rank 0's shard = the config itself)
    digest = {"ok": None, "why": "workload differs from the BASELINE config"}
    if plain and rank == 0:
        digest = check_digest(sim, cfg, a.config, a.steps * sps)

    # ---- end to end through the C ABI with HOST buffers: upload couplings (pinned int8),
    #      run the step, read the energies back
    from ea_inputs import random_couplings
    Jpin = torch.empty((cfg.R, 3, cfg.N), dtype=torch.int8).pin_memory()
    Jpin.numpy()[...] = random_couplings(cfg.R, cfg.N, 1000 + rank)
    Jnp = Jpin.numpy()
    e2e_steps = max(2, min(a.steps, 3))
    sim.set_couplings(Jnp); step(); sim.energy()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        sim.set_couplings(Jnp)
        if me:
            sim.pair_couplings()
        step()
        E = sim.energy()
    barrier()
    e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3, world)
    e2e_value = e2e_ms * 1e9 / (attempts_step * e2e_steps)
    Rp = 32 * cfg.W
    h2d = int(Jnp.nbytes)
    d2h = int(Rp * cfg.n_temps * 4 + Rp * cfg.n_temps)            # energies by slot + sigma
    sim.destroy()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline: the sweep kernel is ALU-pipe bound
    peak = measure_int_peak(torch.cuda.current_stream().cuda_stream)
    # resident / streaming kernel: one launch per step, so the step time IS the kernel's launch
    # duration; generic path: the step is sweep + energy + swap launches and the figure is for the step.
    # second layout: per attempt 5 (Philox XOR3, one call per four sites of ONE replica) + 6 (class of
    # the replica's bit from the three planes) + 2 (64-bit compare) + 2 (flip bit) + 14 / n_temps
    # (bonds and adder, shared by the word's replicas) ALU-pipe lane-ops: x 32 per "word update"
    ops_per_update = 32.0 * (15.0 + 14.0 / cfg.n_temps) if replica else alu_ops_per_update(cfg, sps)
    step_s = float(np.mean(step_ms)) * 1e-3
    achieved = ops_per_update * cfg.n_temps * cfg.W * cfg.N * sps / step_s
    prof = ncu_profile_numbers(a.config) if plain else None
    roofline = {"bound": "alu", "achieved": achieved / 1e12, "peak": peak["lop3"] / 1e12, "unit": "Tlaneop/s",
                "frac": achieved / peak["lop3"], "traffic": prof["dram_bytes"] if prof else None,
                "traffic_source": (prof["file"] + ": dram__bytes_read.sum + dram__bytes_write.sum of one launch "
                                   "(the state is read once per launch whatever the number of sweeps)") if prof else None,
                "ncu_alu_pipe_busy_pct_on_busiest_sm": prof["alu_pipe_max_pct"] if prof else None,
                "note": "ALU-pipe lane-ops: %.1f per word update (DESIGN.md s8) / measured LOP3 issue peak "
                        "(ea_measure_int_peak, same process); IMAD peak %.2f, LOP3+IMAD mix %.2f Tlaneop/s"
                        % (ops_per_update, peak["imad"] / 1e12, peak["mix"] / 1e12)}
    if kernel == 4:
        roofline["hbm_view"] = hbm_view(cfg, sps, step_s)

    per_config = None
    if a.per_config and world == 1 and not replica:
        per_config = per_config_block(torch, EA, flush_l2, peak["lop3"], a.config if plain and sps >= 1000 else None)
        if plain and sps >= 1000:
            ent = {"workload": cfg.name, "kernel": KERNEL_NAMES.get(kernel), "sweeps_per_step": sps,
                   "us_per_sweep": step_s * 1e6 / sps, "ps_per_attempt": value, "alu_frac": roofline["frac"], "digest": digest}
            if kernel == 4:
                ent["hbm_view"] = roofline["hbm_view"]
            ent["oracle_one_core_ps"] = oracle_one_core(cfg)
            per_config[str(a.config)] = ent

    # ---- CPU oracle on the host cores: bounded samples of the same workload, all cores and one core
    cores = len(os.sched_getaffinity(0))
    words = min(cores, cfg.W)
    o_sweeps = max(1, int(4.0e8 / (32 * cfg.n_temps * cfg.N)))     # ~10 s per core
    cpu_ps, cpu_wall = oracle_sample(cfg, words, o_sweeps, words, a.field)
    sample = f"{words} of {cfg.W} words (32 realizations x {cfg.n_temps} temperatures each) x {o_sweeps} sweeps, {cpu_wall:.1f} s wall"
    one_sweeps = max(1, o_sweeps // 2)
    one_ps, one_wall = oracle_sample(cfg, 1, one_sweeps, 1, a.field)

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
        "ms_per_step": total_ms / a.steps, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "u32 bit-sliced words (32 realizations each), u32 Philox draws", "data": "synthetic",
        "config": {"workload": cfg.name, "L": cfg.L, "n_temps": cfg.n_temps, "realizations_per_gpu": cfg.R,
                   "swap_interval": cfg.swap_interval, "sweeps_per_step": sps, "seed": cfg.seed,
                   "field": a.field, "measure_every": me, "layout": a.layout, "swap_mode": a.swap_mode,
                   "kernel": KERNEL_NAMES.get(kernel, str(kernel)),
                   "l2": "flushed between timed steps (256 MiB write); state is re-read from HBM each step",
                   "parallelism": f"shard by realization word x{world}, no collective"},
        "clocks": _clock_summary(samples),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / e2e_steps,
                "what": "ea_set_couplings(host J, pinned) + ea_sweep + ea_energy(host E) per step"},
        "gpu_launches": int(launches),
        "digest_ok": digest["ok"], "digest": digest,
        "roofline": roofline,
        "cpu_baseline": {"value": cpu_ps, "unit": UNIT, "cores": words, "kind": "oracle", "sample": sample,
                         "one_core": {"value": one_ps, "unit": UNIT, "cores": 1,
                                      "sample": f"1 word x {one_sweeps} sweeps, {one_wall:.1f} s wall"}},
        "per_config": per_config,
        "context": {"paper_ps_per_attempt_gtx580": PAPER_PS, "step_ms": step_ms},
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    if digest["ok"] is False:
        print("bench.py: the timed trajectory does NOT match the oracle digest", file=sys.stderr)
        sys.exit(1)


def respawn_under_torchrun(a):
    """`python bench.py --gpus N` without a launcher: build once, then one rank per GPU under
    torch.distributed.run on 127.0.0.1 (the driver's own launch form)."""
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={a.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--sweeps-per-step", type=int, default=5000)
    ap.add_argument("--swap-interval", type=int, default=None,
                    help="override the config's PT cadence (the paper's own benchmark swaps every 10 sweeps, PAPER.md:307)")
    ap.add_argument("--realizations", type=int, default=None,
                    help="override the config's number of disorder realizations per GPU (scaling studies)")
    ap.add_argument("--field", type=int, default=0, help="external field h (SURVEY 8(f2)); default 0 = headline workload")
    ap.add_argument("--measure-every", type=int, default=0,
                    help="accumulate two-copy overlap / energy moments every M sweeps (SURVEY 8(f1)); default off")
    ap.add_argument("--layout", default="realization", choices=["realization", "replica"],
                    help="multispin coding: bits = realizations (BASELINE configs) or the paper's own bits = temperature "
                         "replicas with one random number per replica (SURVEY 8(f3), ea_set_layout)")
    ap.add_argument("--swap-mode", default="permute", choices=["permute", "move"],
                    help="an accepted swap exchanges temperature indices (BASELINE configs) or moves the two lattices "
                         "(SURVEY 8(f3), ea_set_swap_mode)")
    ap.add_argument("--no-per-config", dest="per_config", action="store_false",
                    help="skip the per_config block (ps per attempt of the other BASELINE configs)")
    ap.add_argument("--ref-cores", type=int, default=0, help="--impl reference: processes to use (default: all cores)")
    a = ap.parse_args()
    a.warmup = max(a.warmup, 3) if a.impl == "cuda" else a.warmup
    cfg = CONFIGS[a.config]
    import dataclasses
    if a.swap_interval is not None:
        cfg = dataclasses.replace(cfg, swap_interval=a.swap_interval)
    if a.realizations is not None:
        cfg = dataclasses.replace(cfg, R=a.realizations, name=f"{cfg.name}_R{a.realizations}")
    if a.impl == "reference":
        run_reference(a, cfg)
        return
    # every rank builds under a file lock (a no-op when the library is up to date), so no rank can
    # load a stale or half-written library whatever the launcher's start-up order
    from paper_1311_5582_b200.build import build_library
    build_library()
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(respawn_under_torchrun(a))
    run_cuda(a, cfg)


if __name__ == "__main__":
    main()
