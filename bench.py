#!/usr/bin/env python
"""bench.py -- coupled-pair updates per ns on B200 at L=16384 (BASELINE.json metric), with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C5] [--sweeps-per-step S]

A "step" is one pass of the whole hot path over one batch: S sweeps (default: the whole run of the config; 100 for BASELINE config 5)
of the configured lattice, each sweep = two conflict-free phases of N/4 coupled-pair updates (schedule, loads, Philox,
proposal, dE class, acceptance, write-back, per-sweep observables and their fp64 accumulation).  One process per GPU; with N > 1 every rank runs its own lattice copy (the path shards over replicas,
PAPER.md:141; no data-path collective) and the value is the aggregate over ranks ("weak").

Prints ONE JSON line on rank 0.  `--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores.
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

import ic_inputs  # noqa: E402

METRIC = "coupled-pair updates/ns on 1 B200 and % of HBM roofline (L=16384)"
UNIT = "pair-updates/ns"
B_ALG_PER_PAIR = {8: 4.0, 2: 1.0}     # bytes: every site once in, once out per sweep
B_2PASS_PER_PAIR = {8: 8.0, 2: 2.0}   # two data-dependent phases, each one read + one write of the lattice


def csrc_sha16():
    """Hash of the kernel sources: a profile summary under profiles/ belongs to exactly one state of csrc/."""
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2301_11735_b200", "csrc", "*"))):
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def profiled(config, bits):
    """ncu-derived figures of the dominant kernel (dram bytes and warp instructions per launch) from the newest
    profiles/*_summary.csv written for this config; they are reported only while csrc/ still hashes to the state that was
    profiled, otherwise roofline.traffic is null (a stale capture is not a measurement of this build)."""
    import glob
    best = None
    for f in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_summary.csv"))):
        kv = {}
        for ln in open(f).read().splitlines()[1:]:
            if "," in ln:
                k, v = ln.split(",", 1)
                kv[k.strip()] = v.strip()
        if kv.get("config") == config and int(kv.get("bits", "8")) == bits:
            best = kv
    if not best:
        return None
    best["stale"] = best.get("source_sha16") != csrc_sha16()
    return best


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe): NVML polled from
    a thread every few ms (the timed region is a fraction of a second); nvidia-smi is the fallback."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.rows, self.reasons, self.stop_flag, self.thread, self.proc, self.nvml = index, [], set(), False, None, None, None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.thread = threading.Thread(target=self._poll, daemon=True); self.thread.start()
        except Exception:
            self.nvml = None
            try:
                self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                              "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
                self.thread = threading.Thread(target=self._read, daemon=True); self.thread.start()
            except Exception:
                self.proc = None

    def _poll(self):
        n = self.nvml
        bits = [("hw_slowdown", getattr(n, "nvmlClocksEventReasonHwSlowdown", 0x8)),
                ("hw_thermal_slowdown", getattr(n, "nvmlClocksEventReasonHwThermalSlowdown", 0x40)),
                ("sw_thermal_slowdown", getattr(n, "nvmlClocksEventReasonSwThermalSlowdown", 0x20)),
                ("sw_power_cap", getattr(n, "nvmlClocksEventReasonSwPowerCap", 0x4))]
        get_reasons = getattr(n, "nvmlDeviceGetCurrentClocksEventReasons", None) or getattr(n, "nvmlDeviceGetCurrentClocksThrottleReasons")
        while not self.stop_flag:
            try:
                mhz = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
                pw = n.nvmlDeviceGetPowerUsage(self.handle) / 1000.0
                self.rows.append((mhz, pw))
                r = int(get_reasons(self.handle))
                for name, bit in bits:
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def _read(self):
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.proc.stdout:
            c = [x.strip() for x in ln.split(",")]
            if len(c) >= 7 and c[0].replace(".", "").isdigit():
                self.rows.append((float(c[0]), float(c[2]) if c[2].replace(".", "").isdigit() else 0.0))
                self.max_mhz = float(c[1]) if c[1].replace(".", "").isdigit() else None
                for k, nme in enumerate(names):
                    if c[3 + k].lower().startswith("active"):
                        self.reasons.add(nme)

    def stop(self):
        if self.thread is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no NVML and no nvidia-smi"]}
        self.stop_flag = True
        if self.proc:
            time.sleep(0.05); self.proc.terminate()
        self.thread.join(timeout=2)
        sm = sorted(r[0] for r in self.rows)
        pw = [r[1] for r in self.rows]
        order = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": getattr(self, "max_mhz", None),
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": [r for r in order if r in self.reasons],
                "source": "nvml" if self.nvml else "nvidia-smi"}


def cpu_oracle_rate(cfg, code, nsweeps, threads):
    """Pair updates per ns of the CPU oracle (oracle/ic_oracle.c, as it stands) on `nsweeps` sweeps of `code`."""
    import oracle
    lat = oracle.Lattice(code, cfg["delta"], cfg["V"], cfg["J"], cfg["seed"])
    t0 = time.perf_counter()
    lat.sweep_s1(cfg["T"][0], nsweeps, threads=threads)
    dt = time.perf_counter() - t0
    return (code.size // 2) * nsweeps / (dt * 1e9), dt


def run_reference(args, cfg):
    """Reference arm = the CPU oracle on the host cores; each step is a bounded sample: 1 sweep of a 4096 x 4096 corner
    of the workload's lattice shape (same parameters, same charge density), all cores."""
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    Ls = min(cfg["L"], 4096)
    dens = cfg["nplus"] / float(cfg["L"]) ** 2
    code = oracle.init_state(Ls, Ls, int(round(dens * Ls * Ls)), 0, cfg["seed"], 0)
    lat = oracle.Lattice(code, cfg["delta"], cfg["V"], cfg["J"], cfg["seed"])
    for _ in range(args.warmup):
        lat.sweep_s1(cfg["T"][0], 1, threads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        lat.sweep_s1(cfg["T"][0], 1, threads=cores)
    dt = time.perf_counter() - t0
    pairs = (Ls * Ls // 2) * args.steps
    val = pairs / (dt * 1e9)
    sample = f"1 sweep per step of a {Ls}x{Ls} lattice with the workload's parameters and charge density ({pairs} pair updates timed)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": f"{args.config}: L={cfg['L']} n={cfg['n']} Delta={cfg['delta']} V={cfg['V']} J={cfg['J']} T={cfg['T'][0]}",
                   "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "site_updates_per_s": 2e9 * val,
    }), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C5", choices=sorted(ic_inputs.CONFIGS))
    ap.add_argument("--sweeps-per-step", type=int, default=0, help="0 = the sweeps of the config's whole run (C5: 100)")
    ap.add_argument("--bits", type=int, default=0, help="override bits per site (8 or 2)")
    ap.add_argument("--variant", type=int, default=0, help="kernel variant (0 = automatic)")
    ap.add_argument("--replicas", type=int, default=0, help="override the number of lattice copies per GPU (temperatures repeat cyclically): "
                    "with >= 4 x the SM count a small-lattice config shows its saturated rate instead of its latency-bound one")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target duration of the timed CPU-oracle sample")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    cfg = dict(ic_inputs.CONFIGS[args.config])
    if args.bits:
        cfg["bits"] = args.bits
    if args.replicas > 0:
        cfg["T"] = [cfg["T"][i % len(cfg["T"])] for i in range(args.replicas)]
    if args.sweeps_per_step <= 0:
        args.sweeps_per_step = int(cfg["sweeps"])
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import torch.distributed as dist

    import paper_2301_11735_b200 as ic
    from paper_2301_11735_b200 import shard

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1")); local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    L, Ts, bits, S = cfg["L"], cfg["T"], cfg["bits"], args.sweeps_per_step
    reps = len(Ts)
    N = L * L
    # every rank owns `reps` lattice copies of its own: same parameters, seed offset by the rank (weak scaling over replicas)
    sim = ic.Sim(L, cfg["n"], cfg["delta"], cfg["V"], cfg["J"], seed=cfg["seed"] + 1000 * rank, replicas=reps, bits_per_site=bits)
    if cfg["nminus"]:
        for r in range(reps):
            sim.init_charges(r, cfg["nplus"], cfg["nminus"])
    if args.variant:
        sim.set_variant(args.variant)
    assert sim.Q == cfg["nplus"] - cfg["nminus"]
    pairs_per_step = reps * (N // 2) * S

    # ---- device-resident throughput -------------------------------------------------------------------------------
    for _ in range(args.warmup):
        sim.sweep(Ts, S)
    barrier()
    sampler = ClockSampler(local); sampler.start()
    l0 = sim.launch_count
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        sim.sweep(Ts, S)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = sim.launch_count - l0
    clocks = sampler.stop()
    ms = shard.max_over_ranks(ms)                      # a multi-rank time is the slowest rank's
    value = world * pairs_per_step * args.steps / (ms * 1e6)

    # invariants after the timed region: eq. (2) and incremental == recomputed integers
    obs = sim.observables()
    for r in range(min(reps, 2)):
        assert list(sim.debug_recompute(r)) == [obs[r][k] for k in ("n2", "bV", "bJ", "M", "Ms", "Q")], "integers drifted"
        assert obs[r]["Q"] == sim.Q
    # the job's lattice copies are the world * reps global replicas, dealt round-robin (shard.replica_shard); the one
    # exchange of the whole job is this gather of about 100 B per replica
    mine = shard.replica_shard(world * reps, rank, world)
    all_obs = shard.gather_observables({g: {k: obs[i][k] for k in ("Q", "nmeas", "n2", "bV", "bJ", "M", "Ms")} for i, g in enumerate(mine)},
                                       world * reps)
    assert all(o["Q"] == sim.Q and o["nmeas"] == obs[0]["nmeas"] for o in all_obs), "a rank lost charge or sweeps"

    # ---- end to end through the C ABI with HOST buffers ----------------------------------------------------------------
    e2e = None
    if not args.no_e2e:
        host_in = torch.empty((reps, N), dtype=torch.int8).pin_memory()
        host_out = torch.empty((reps, N), dtype=torch.int8).pin_memory()
        for r in range(reps):
            sim.state(r, out=host_in[r])
        e2e_steps = max(1, min(args.steps, 3))
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            for r in range(reps):
                sim.set_state(r, host_in[r])          # H2D of the step's input lattice (validated, eq. 2)
            sim.sweep(Ts, S)
            for r in range(reps):
                sim.state(r, out=host_out[r])         # D2H of the result lattice
            o = sim.observables()                     # D2H of the step's observables
        barrier()
        dt = time.perf_counter() - t0
        dt = shard.max_over_ranks(dt)
        e2e = {"value": world * pairs_per_step * e2e_steps / (dt * 1e9), "unit": UNIT,
               "h2d_bytes_per_step": reps * N + 8 * reps, "d2h_bytes_per_step": reps * N + 128 * reps, "steps": e2e_steps,
               "path": "ic_set_state(pinned host) -> ic_sweep -> ic_state(pinned host) + ic_observables"}

    # ---- the same with the host lattices at 2 bits per site (ic_set_state_packed / ic_state_packed): a quarter of the PCIe bytes
    e2e_packed = None
    if not args.no_e2e:
        del host_in, host_out
        pk_in = torch.empty((reps, N // 4), dtype=torch.uint8).pin_memory()
        pk_out = torch.empty((reps, N // 4), dtype=torch.uint8).pin_memory()
        for r in range(reps):
            sim.state_packed(r, out=pk_in[r])
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            for r in range(reps):
                sim.set_state_packed(r, pk_in[r])     # H2D of the step's input lattice, 2 bits per site (eq. 2 checked on the device)
            sim.sweep(Ts, S)
            for r in range(reps):
                sim.state_packed(r, out=pk_out[r])    # D2H of the result lattice, 2 bits per site
            o = sim.observables()
        barrier()
        dt = shard.max_over_ranks(time.perf_counter() - t0)
        e2e_packed = {"value": world * pairs_per_step * e2e_steps / (dt * 1e9), "unit": UNIT,
                      "h2d_bytes_per_step": reps * N // 4 + 8 * reps, "d2h_bytes_per_step": reps * N // 4 + 128 * reps, "steps": e2e_steps,
                      "path": "ic_set_state_packed(pinned host, 2 bits/site) -> ic_sweep -> ic_state_packed(pinned host) + ic_observables"}

    # ---- roofline of the dominant kernel (one phase launch = N/4 pair updates per replica) ----------------------------------
    peak, peak_src = measured_peaks()
    phase_launches = 2 * S * args.steps
    avg_ms = ms / phase_launches                     # the per-sweep fold kernel (1 thread per replica) is inside this average
    pairs_per_launch = reps * N // 4
    ach = B_ALG_PER_PAIR[bits] * pairs_per_launch / (avg_ms * 1e6)
    ach2 = B_2PASS_PER_PAIR[bits] * pairs_per_launch / (avg_ms * 1e6)
    prof = profiled(args.config, bits) if world == 1 else None
    roofline = {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": float(prof["dram_bytes_per_launch"]) if prof and not prof["stale"] else None,
                "traffic_source": (f"profiles/{prof['profile']}_summary.csv" + (" (stale: csrc/ changed since that capture)" if prof["stale"] else "")) if prof else None,
                "kernel": "phase kernel (one of the two phases of a sweep)", "avg_launch_ms": avg_ms, "peak_source": peak_src,
                "bytes_per_pair_algorithmic": B_ALG_PER_PAIR[bits],
                "two_pass": {"bytes_per_pair": B_2PASS_PER_PAIR[bits], "achieved": ach2, "frac": ach2 / peak}}

    if prof and not prof["stale"]:
        ipp = float(prof["instructions_per_pair"])
        mhz = clocks.get("sm_mhz") or 1965.0
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        issue_peak = sms * 4 * 32 * mhz * 1e6       # one warp instruction per cycle and sub-partition
        roofline["issue"] = {"what": "lane-instructions issued per second against one warp instruction per cycle and SM sub-partition; "
                                     "the capture shows the shared-memory data pipe as the busiest unit",
                             "achieved": value * 1e9 * ipp, "peak": issue_peak, "unit": "lane-instructions/s",
                             "frac": value * 1e9 * ipp / issue_peak, "instructions_per_pair": ipp, "sm_count": sms,
                             "lsu_data_pipe_pct_in_capture": float(prof.get("lsu_data_pipe_wavefronts_pct", "nan"))}
    out = None
    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8" if bits == 8 else "u2", "data": "synthetic",
            "config": {"arithmetic": f"{'1 byte' if bits == 8 else '2 bits'} per site, uint32 Philox words and thresholds, int64 / fp64 observables",
                       "workload": f"{args.config}: L={L} n={cfg['n']} Delta={cfg['delta']} V={cfg['V']} J={cfg['J']} "
                                   f"T={Ts[0]}..{Ts[-1]} x{reps} replica(s), {bits} bits/site, seeded stage-1 state with exact charge {sim.Q}",
                       "sweeps_per_step": S, "pairs_per_step_per_gpu": pairs_per_step, "parallelism": f"replicas x{world}",
                       "l2": f"lattice {reps * N * bits // 8 >> 20} MiB per GPU " + ("> 126 MB L2 (inputs larger than L2, no flush)" if reps * N * bits // 8 > 126e6 else "fits L2 (L2-resident by design)")},
            "site_updates_per_s": 2e9 * value, "clocks": clocks, "gpu_launches": launches, "roofline": roofline,
        }
        if e2e:
            out["e2e"] = e2e
            out["e2e_packed"] = e2e_packed
        if world == 1 and not args.no_cpu_baseline:
            cores = os.cpu_count() or 1
            Ls = min(L, 8192)
            import oracle
            dens = cfg["nplus"] / float(N)
            code = oracle.init_state(Ls, Ls, int(round(dens * Ls * Ls)), 0, cfg["seed"], 0)
            nsw = max(1, int(args.cpu_seconds * 0.07e9 * min(cores, 16) / 16 / (Ls * Ls // 2)))   # ~0.07 pairs/ns on 16 cores
            v, dt = cpu_oracle_rate(cfg, code, nsw, cores)
            out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
                                   "sample": f"{nsw} sweeps of a {Ls}x{Ls} lattice with the workload's parameters and charge density, OpenMP over rows"}
    sim.close()
    if world > 1:
        dist.barrier(); dist.destroy_process_group()
    if out:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
