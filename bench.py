#!/usr/bin/env python
"""bench.py -- throughput of the population-annealing hot path on B200 (contract in the task prompt).

    python bench.py --gpus 1 --steps K --warmup W            # this library, one JSON line
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on the host cores
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

Default workload: BASELINE.json configs[4] (cfg5: L=256, R=10^6, 8.2 GB of packed spins), the largest single-GPU
configuration; the others are carried as compact sub-records (`other_configs`), `--config N` makes any of them the main line.

A "step" is one temperature step of PAPER.md Sec. 2.1 (L56-L62) over one synthetic population:
resample beta_{i-1} -> beta_i (energies, weights, TREE1024 normaliser, copy numbers, prefix sum,
replica copy), theta checkerboard Metropolis sweeps at beta_i, energies + observables
(+ multi-histogram accumulation where the workload asks for it).  metric = spin updates per ns.

N > 1: the path shards as independent populations ("replicas only"): every rank
anneals its own population (seed + rank) with no data-path collective; weak scaling.
"""
import argparse
import ctypes
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1703_03676_b200.workloads import CONFIGS  # noqa: E402

METRIC = "spin_updates_per_ns"
UNIT = "updates/ns"
# Algorithmic work of the dominant kernel (the sweep): 131 IMAD.WIDE.U32 per word of
# 32 spins (8 Philox4x32-10 calls sharing rounds 1-3) = 4.09375 wide multiplies per spin update; the
# FMA-heavy pipe issues 32 of them per clock per SM on 148 SMs.
WIDE_MUL_PER_UPDATE = 131.0 / 32.0
WIDE_MUL_PER_CLK_PER_SM = 32.0
N_SM_FALLBACK = 148            # B200; used only where no CUDA device can be asked (the reference arm never needs it)
_n_sm = None


def n_sm():
    """SM count of the current device (the roofline peaks scale with it)."""
    global _n_sm
    if _n_sm is None:
        try:
            import torch
            _n_sm = int(torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count)
        except Exception:
            _n_sm = N_SM_FALLBACK
    return _n_sm


LCG_INSTR_PER_UPDATE = 5.0
ISSUE_LANES_PER_CLK_PER_SM = 128.0

def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """SM clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe).  NVML is polled from a thread every
    2 ms (the timed region of the small configs is tens of milliseconds: `nvidia-smi -lms` is too coarse for it); if NVML
    cannot be loaded the recipe's nvidia-smi loop is the fallback."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.nv, self.stop_flag, self.thread = index, [], None, None, False, None
        self.sm, self.reasons, self.mx = [], set(), None

    def _nvml_index(self, nv):
        # CUDA_VISIBLE_DEVICES remaps CUDA ordinals; find the NVML handle of the CUDA device by UUID
        import torch
        try:
            uuid = str(torch.cuda.get_device_properties(self.index).uuid)
            for i in range(nv.nvmlDeviceGetCount()):
                h = nv.nvmlDeviceGetHandleByIndex(i)
                u = nv.nvmlDeviceGetUUID(h)
                u = u.decode() if isinstance(u, bytes) else u
                if uuid in u:
                    return h
        except Exception:
            pass
        return nv.nvmlDeviceGetHandleByIndex(self.index)

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            self.nv, self.h = nv, self._nvml_index(nv)
            self.mx = float(nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM))
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nv = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _poll(self):
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0)),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0)),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0)),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0))}
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", getattr(nv, "nvmlDeviceGetCurrentClocksThrottleReasons", None))
        while not self.stop_flag:
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                if get_reasons is not None:
                    r = int(get_reasons(self.h))
                    for n, bit in names.items():
                        if bit and (r & bit):
                            self.reasons.add(n)
            except Exception:
                pass
            time.sleep(0.002)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.nv is not None:
            self.stop_flag = True
            self.thread.join(timeout=1)
            sm = self.sm
            busy = [c for c in sm if self.mx and c > 0.5 * self.mx] or sm
            return {"sm_mhz": statistics.median(busy) if busy else None, "sm_max_mhz": self.mx, "reasons": sorted(self.reasons),
                    "samples": len(sm), "source": "NVML polled every 2 ms during the timed region"}
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
                for n, v in zip(names, r[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        busy = [c for c in sm if mx and c > 0.5 * max(mx)] or sm
        return {"sm_mhz": statistics.median(busy) if busy else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "source": "nvidia-smi -lms 100"}


def reduce_over_ranks(ms, units, device, dist=None):
    """N > 1 (replicas only): the job's time is the MAX over ranks, its work the SUM over ranks.
    `dist` = torch.distributed when a process group is up (nccl on the GPU box, gloo in tests/test_multirank_gloo.py)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms), float(units)
    import torch
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


COMBINE_KEYS = ("e", "C", "absm", "m2", "m4")


def combine_over_ranks(lnZ, obs, device, dist, wavg):
    """The one exchange step the method has across independent populations (Sec. 2.2, Eq. 6-7):
    all-gather (lnZ_m, observables_m) -- 6 doubles per rank -- and weight run m by exp(-beta F_m) = exp(lnZ_m).
    `wavg(lnZ[M], A[M][nobs]) -> (A~, omega)` is the library's pa_weighted_average (the oracle's in the CPU test)."""
    import torch
    mine = torch.tensor([float(lnZ)] + [float(obs[k]) for k in COMBINE_KEYS], dtype=torch.float64, device=device)
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        rows = mine[None, :].cpu().numpy()
    else:
        buf = [torch.empty_like(mine) for _ in range(dist.get_world_size())]
        dist.all_gather(buf, mine)
        rows = torch.stack(buf).cpu().numpy()
    out, omega = wavg(rows[:, 0].copy(), rows[:, 1:].copy())
    return {"runs": int(rows.shape[0]), "omega": [float(x) for x in omega], **{k: float(v) for k, v in zip(COMBINE_KEYS, out)}}


def rank_seed(wl, rank):
    """Every rank anneals its own independent population (no data-path collective)."""
    return wl.seed + rank


def one_step(pop, wl, beta_prev, beta, fused=False):
    if fused and not wl.multi_histogram:
        return pop.anneal([beta_prev, beta], wl.theta)[0]              # the same step through pa_anneal: no host round trip inside
    pop.resample(beta_prev, beta)
    pop.sweep(beta, wl.theta)
    obs = pop.observables(beta)
    if wl.multi_histogram:
        pop.hist_accumulate(beta)
    return obs


def first_run_decides(d, dist):
    """PAPER.md L118 (Sec. 2.3): "our code used in adaptive mode decides about temperature steps only in the first run and keeps
    the temperature sequence fixed for the remaining passes" -- the condition under which Eq. 6-7 may average the runs at every
    temperature.  With one run per rank the first run is rank 0: it alone bisects (`d` = its step, None on the other ranks) and its
    8-byte step is broadcast; it is part of the temperature step and sits inside the timed region."""
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(d) if dist.get_rank() == 0 else 0.0], dtype=torch.float64, device=dev)
    dist.broadcast(t, src=0)
    return float(t.item())


def next_beta(pop, wl, betas, i, beta_prev, dist=None):
    if wl.n_steps is not None:
        return betas[min(i, len(betas) - 1)]
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        d = first_run_decides(pop.adapt_dbeta(wl.target_overlap, beta_prev, wl.beta_f) if dist.get_rank() == 0 else None, dist)
    else:
        d = pop.adapt_dbeta(wl.target_overlap, beta_prev, wl.beta_f)
    return min(wl.beta_f, beta_prev + d)


def whole_run(pa, wl, seed, rng):
    """the config's WHOLE annealing schedule on a fresh population, timed as the paper times its runs:
    t_SF = t_run / (N theta sum_i R_i) (Eq. 11), resampling, measurement (and, for the adaptive config, the
    bisection and the histogram fold) included; the resample cost depends on the weight distribution, so it is sampled in
    situ at every step (median, max, and near beta = 0.1, beta_c, the last step), as is the sweep kernel's rate.  The in-situ
    phase events cost time on a stream of small kernels, so where a run takes seconds it is done twice: once with the default
    timing (sweep only) for t_SF, once instrumented for the per-step figures."""
    import torch

    def run(mask):
        pop = pa.Population(wl.L, wl.R, seed, dims=wl.dims)
        pop.set_timing(mask)
        if rng == "lcg":
            pop.set_rng_mode(pa.PA_RNG_LCG)
        betas = wl.betas() if wl.n_steps is not None else None
        beta_prev, i = wl.beta0, 0
        obs = pop.observables(beta_prev)
        if wl.multi_histogram:
            pop.hist_accumulate(beta_prev)
        rows, flips = [], 0
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        while beta_prev < wl.beta_f and (betas is None or i < len(betas) - 1):
            i += 1
            beta = next_beta(pop, wl, betas, i, beta_prev)
            obs = one_step(pop, wl, beta_prev, beta)
            flips += obs["R"] * wl.N * wl.theta
            if mask & pa.PA_TIME_RESAMPLE:
                rt, ct = pop.last_resample_ms()
                rows.append((beta, obs["R"] * wl.N * wl.theta / (pop.last_sweep_ms() * 1e6), rt, ct))
            beta_prev = beta
        torch.cuda.synchronize()
        t_run = time.perf_counter() - t0
        pop.close()
        return t_run, flips, rows, obs, beta_prev, i

    full = pa.PA_TIME_SWEEP | pa.PA_TIME_RESAMPLE
    twice = wl.R * wl.N <= 2 * 10**9                                   # cfgs 1-4: seconds; cfg5: minutes, one instrumented pass
    t_run, flips, rows, obs, beta_last, nsteps = run(pa.PA_TIME_SWEEP if twice else full)
    if twice:
        _, _, rows, _, _, _ = run(full)
    betas = wl.betas() if wl.n_steps is not None else None

    def near(b):
        return min(rows, key=lambda r: abs(r[0] - b))
    res = sorted(r[2] for r in rows)
    marks = {"beta_0.1": near(0.1), "beta_c": near(0.4406868), "last": rows[-1]}
    out = {"steps": nsteps, "beta_final": beta_last, "t_run_s": t_run, "t_SF_ns": t_run * 1e9 / flips, "updates_per_ns": flips / (t_run * 1e9),
           "timing": "host wall clock around the whole schedule, synchronised on both sides (the paper's t_SF, Eq. 11)"
                     + ("; per-step figures from a second, instrumented run" if twice else ""),
           "resample_ms": {"median": res[len(res) // 2], "max": res[-1], **{k: v[2] for k, v in marks.items()}},
           "sweep_updates_per_ns": {k: v[1] for k, v in marks.items()},
           "final_observables": obs}
    if wl.n_steps is not None and not wl.multi_histogram:
        # the same schedule in ONE pa_anneal call (no host round trip between its steps); a two-step call on a throw-away
        # population first, so that the one-time costs of the first pa_anneal of a process (pinned staging, lazy kernel loading: 20 ms)
        # stay outside the clock, as they do for the single calls (warmed by the timed steps before the whole run)
        warm = pa.Population(wl.L, wl.R, seed, dims=wl.dims)
        if rng == "lcg":
            warm.set_rng_mode(pa.PA_RNG_LCG)
        warm.anneal(betas[:3], wl.theta)
        warm.close()
        pop = pa.Population(wl.L, wl.R, seed, dims=wl.dims)
        pop.set_timing(0)
        if rng == "lcg":
            pop.set_rng_mode(pa.PA_RNG_LCG)
        pop.observables(wl.beta0)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        obs2 = pop.anneal(betas, wl.theta)
        t2 = time.perf_counter() - t0
        flips2 = sum(o["R"] for o in obs2) * wl.N * wl.theta
        out["one_call"] = {"api": "pa_anneal", "t_run_s": t2, "t_SF_ns": t2 * 1e9 / flips2, "updates_per_ns": flips2 / (t2 * 1e9),
                           "same_final_observables": obs2[-1] == obs}
        pop.close()
    return out


def theta_scan(args):
    """PAPER.md Table 3 (t_SF against theta at L = 128, R = 50 000), Table 4 (fraction of the run time spent in the spin-update
    kernel) re-measured on this GPU: whole runs, host wall clock.  Context for BASELINE.md, not the bench line."""
    import torch
    from paper_1703_03676_b200 import pa
    from paper_1703_03676_b200.workloads import table3_workload
    torch.cuda.set_device(0)
    rows = []
    # one-time costs of the process (lazy kernel loading, pinned staging of the first pa_anneal) stay outside the clocks
    wl = table3_workload(1)
    warm = pa.Population(wl.L, wl.R, wl.seed)
    if args.rng == "lcg":
        warm.set_rng_mode(pa.PA_RNG_LCG)
    wb = wl.betas()
    warm.observables(wb[0])
    one_step(warm, wl, wb[0], wb[1])
    warm.anneal(wb[1:4], 1)
    warm.close()
    for theta in (1, 5, 10, 50, 100, 500):
        wl = table3_workload(theta)
        pop = pa.Population(wl.L, wl.R, wl.seed)
        if args.rng == "lcg":
            pop.set_rng_mode(pa.PA_RNG_LCG)
        betas = wl.betas()
        pop.observables(betas[0])
        flips, sweep_ms = 0, 0.0
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for i in range(1, len(betas)):
            obs = one_step(pop, wl, betas[i - 1], betas[i])
            flips += obs["R"] * wl.N * theta
            sweep_ms += pop.last_sweep_ms()
        torch.cuda.synchronize()
        t_run = time.perf_counter() - t0
        pop.close()
        # the same run in one pa_anneal call
        pop = pa.Population(wl.L, wl.R, wl.seed)
        pop.set_timing(0)
        if args.rng == "lcg":
            pop.set_rng_mode(pa.PA_RNG_LCG)
        pop.observables(betas[0])
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        obs2 = pop.anneal(betas, theta)
        t2 = time.perf_counter() - t0
        flips2 = sum(o["R"] for o in obs2) * wl.N * theta
        rows.append({"theta": theta, "t_SF_ns": t_run * 1e9 / flips, "updates_per_ns": flips / (t_run * 1e9),
                     "sweep_kernel_fraction": sweep_ms * 1e-3 / t_run, "t_run_s": t_run,
                     "one_call": {"t_SF_ns": t2 * 1e9 / flips2, "updates_per_ns": flips2 / (t2 * 1e9)}})
        pop.close()
    print(json.dumps({"theta_scan": rows, "workload": "PAPER.md Table 3/4 shape: L=128, R=50000, 50 equal steps to beta=1", "rng": args.rng}), flush=True)


def sweep_traffic(wl_name, rng):
    """roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum of ONE sweep launch, read from the tracked ncu export
    profiles/traffic_<workload>_<rng>.csv (the raw page of an `ncu --set full` capture of this bench command, restricted to the
    two counters, base units; the command is in the .md beside it).  None if this workload has no capture."""
    import csv
    import hashlib
    import re
    path = os.path.join(ROOT, "profiles", f"traffic_{wl_name}_{rng}.csv")
    if not os.path.exists(path):
        return None, None
    # the .md beside the export records the sha256 of the sweep kernels' source at capture time: a capture of other code is not
    # this code's traffic
    note = path[:-4] + ".md"
    src = os.path.join(ROOT, "paper_1703_03676_b200", "csrc", "pa_sweep.cu")
    want = re.search(r"sha256\(paper_1703_03676_b200/csrc/pa_sweep\.cu\)\s*=\s*([0-9a-f]{64})", open(note).read()) if os.path.exists(note) else None
    have = hashlib.sha256(open(src, "rb").read()).hexdigest() if os.path.exists(src) else None
    if want is None or have != want.group(1):
        return None, "stale: " + os.path.relpath(path, ROOT) + " was captured on another pa_sweep.cu (sha256 differs or is not recorded)"
    rows = list(csv.reader(open(path)))
    hdr = rows[0]
    try:
        ir, iw, ik = hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum"), hdr.index("Kernel Name")
    except ValueError:
        return None, None
    vals = [float(r[ir]) + float(r[iw]) for r in rows[2:] if len(r) > max(ir, iw) and "pa_sweep" in r[ik]]
    if rows[1][ir] != "byte" or not vals:
        return None, None
    return sum(vals) / len(vals), os.path.relpath(path, ROOT)


def sweep_roof(rng, sm_max):
    """(algorithmic units per update, peak in G units/s, unit, kernel name) of the sweep kernel's binding resource (DESIGN.md 6.1 / 6.4)."""
    if rng == "lcg":
        return LCG_INSTR_PER_UPDATE, n_sm() * ISSUE_LANES_PER_CLK_PER_SM * sm_max * 1e-3, "G thread-instructions/s", "pa_sweep_lcg_kernel"
    return WIDE_MUL_PER_UPDATE, n_sm() * WIDE_MUL_PER_CLK_PER_SM * sm_max * 1e-3, "G IMAD.WIDE.U32/s", "pa_sweep_col_kernel (pa_sweep3d_kernel on a box)"


class Runner:
    """One population of a workload and the bookkeeping of its annealing schedule (which beta comes next)."""

    def __init__(self, pa, wl, seed, rng, couplings="ferro", dims=2, dist=None):
        self.pa, self.wl, self.rng, self.dist = pa, wl, rng, dist
        self.pop = pa.Population(wl.L, wl.R, seed, dims=wl.dims)
        if rng == "lcg":
            self.pop.set_rng_mode(pa.PA_RNG_LCG)
        if couplings == "pmj":
            from paper_1703_03676_b200.workloads import random_couplings
            self.pop.set_couplings(*random_couplings(wl.L, wl.seed))
        self.betas = wl.betas() if wl.n_steps is not None else None
        self.beta, self.i = wl.beta0, 0
        self.pop.observables(self.beta)
        if wl.multi_histogram:
            self.pop.hist_accumulate(self.beta)

    def left(self):
        return 10**9 if self.betas is None else len(self.betas) - 1 - self.i

    def step(self, fused=False):
        """One temperature step (for the adaptive workload the bisection is part of it).  Returns the observables."""
        self.i += 1
        beta = next_beta(self.pop, self.wl, self.betas, self.i, self.beta, self.dist)
        obs = one_step(self.pop, self.wl, self.beta, beta, fused)
        self.beta = beta
        return obs

    def close(self):
        self.pop.close()


def timed_steps(torch, run, K, Wm, flush, fused=False, sampler=None, barrier=None):
    """W warm-up steps, then K timed steps: CUDA events on the library's stream (= torch's current stream) around every step,
    an L2 flush between steps outside the events.  Returns the raw per-rank numbers."""
    wl, pop = run.wl, run.pop
    for _ in range(Wm):
        run.step(fused)
    torch.cuda.synchronize()
    if barrier:
        barrier()
    if sampler:
        sampler.start()
    launches0 = pop.launch_count
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    updates, sweep_ms, sweep_updates, obs = 0, [], [], None
    for s in range(K):
        flush.zero_()                                                          # L2 flush, outside the timed events
        ev[s][0].record()
        obs = run.step(fused)
        ev[s][1].record()
        u = obs["R"] * wl.N * wl.theta
        updates += u
        sweep_ms.append(pop.last_sweep_ms()); sweep_updates.append(u)
    torch.cuda.synchronize()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    return {"total_ms": total_ms, "updates": updates, "sweep_ms": sweep_ms, "sweep_updates": sweep_updates, "obs": obs,
            "launches": pop.launch_count - launches0}


def instrumented_steps(run, n, peaks):
    """SURVEY 8(d), resample: a few more steps with every phase event on (they cost ~3 us each, so they are off in the timed
    region).  Copy kernel against HBM (2 x population bytes), and the whole non-sweep part of a step -- resample chain +
    energies / observables pass -- against its floor of 3 ceil(R/32) N 4 + 24 R bytes."""
    pa, wl, pop = run.pa, run.wl, run.pop
    pop.set_timing(pa.PA_TIME_SWEEP | pa.PA_TIME_RESAMPLE | pa.PA_TIME_MEASURE)
    res, cop, mea, cbytes, fbytes = [], [], [], [], []
    for _ in range(n):
        if run.left() < 1:
            break
        R_old = pop.population
        o = run.step()
        t, c = pop.last_resample_ms()
        res.append(t); cop.append(c); mea.append(pop.last_measure_ms())
        G_new, G_old = (o["R"] + 31) // 32, (R_old + 31) // 32
        cbytes.append(2 * G_new * wl.N * 4)
        fbytes.append((2 * G_new + G_new) * wl.N * 4 + 24 * max(R_old, o["R"]))
    pop.set_timing(pa.PA_TIME_SWEEP)
    if not res:
        return None
    m = lambda v: sum(v) / len(v)                                             # noqa: E731
    hbm = float(peaks["hbm_gbs"])
    cms, rm = m(cop), m(res) + m(mea)
    return {"ms_per_step": m(res), "copy_kernel_ms": cms, "measure_kernel_ms": m(mea),
            "copy_gbs": m(cbytes) / (cms * 1e6), "copy_frac_of_hbm": m(cbytes) / (cms * 1e6) / hbm,
            "resample_plus_measure_ms": rm, "floor_bytes": m(fbytes), "floor_ms": m(fbytes) / (hbm * 1e6),
            "resample_plus_measure_gbs": m(fbytes) / (rm * 1e6), "resample_plus_measure_frac_of_hbm": m(fbytes) / (rm * 1e6) / hbm,
            "hbm_peak_gbs": hbm, "steps": len(res),
            "what": "copy: 2 x packed population bytes / copy kernel time; resample+measure: (3 ceil(R/32) N 4 + 24 R) bytes / "
                    "(pa_resample + energy/observable kernel) time; phase events on, after the timed region"}


def roofline_of(rng, wl_name, sweep_ms, sweep_updates, total_ms, peaks, peak_src):
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    per_upd, peak, unit, kname = sweep_roof(rng, sm_max)
    k_ms, k_upd = sum(sweep_ms) / len(sweep_ms), sum(sweep_updates) / len(sweep_updates)
    achieved = per_upd * k_upd / (k_ms * 1e6)
    traffic, tsrc = sweep_traffic(wl_name, rng)
    per_clk = ISSUE_LANES_PER_CLK_PER_SM if rng == "lcg" else WIDE_MUL_PER_CLK_PER_SM
    return {"bound": "alu", "kernel": kname, "achieved": achieved, "peak": peak, "unit": unit, "frac": achieved / peak,
            "traffic": traffic, "traffic_source": tsrc, "algorithmic_bytes_per_launch": None,
            "peak_source": f"{n_sm()} SM x {per_clk:.0f}/clk/SM x {sm_max:.0f} MHz ({peak_src} sm_max_mhz; DESIGN.md Sec. 6)",
            "kernel_ms": k_ms, "kernel_updates_per_ns": k_upd / (k_ms * 1e6), "share_of_step": sum(sweep_ms) / total_ms,
            "algorithmic_per_update": per_upd}


def sub_record(torch, pa, cfg, rng, flush, peaks, peak_src, K=5, Wm=3):
    """A compact record of another configuration (a few steps): the small-population story and the LCG-assisted stream stay visible
    next to the headline workload."""
    wl = CONFIGS[cfg]
    run = Runner(pa, wl, wl.seed, rng)
    try:
        t = timed_steps(torch, run, K, Wm, flush)
        roof = roofline_of(rng, wl.name, t["sweep_ms"], t["sweep_updates"], t["total_ms"], peaks, peak_src)
        ins = instrumented_steps(run, 3, peaks)
        rec = {"workload": wl.name, "rng": rng, "steps": K, "warmup": Wm, "value": t["updates"] / (t["total_ms"] * 1e6),
               "ms_per_step": t["total_ms"] / K, "gpu_launches": t["launches"],
               "roofline": {k: roof[k] for k in ("frac", "kernel_updates_per_ns", "share_of_step", "kernel_ms", "traffic")},
               "resample": None if ins is None else {k: ins[k] for k in ("ms_per_step", "copy_kernel_ms", "measure_kernel_ms",
                                                                          "copy_frac_of_hbm", "resample_plus_measure_frac_of_hbm")}}
        if wl.n_steps is not None and not wl.multi_histogram and wl.R * wl.N <= 10**9:
            # the launch-bound configurations also through pa_anneal (one call per step: no host round trip inside a step)
            tf = timed_steps(torch, run, K, 1, flush, fused=True)
            rec["pa_anneal_per_step"] = {"value": tf["updates"] / (tf["total_ms"] * 1e6), "ms_per_step": tf["total_ms"] / K}
        return rec
    finally:
        run.close()


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1703_03676_b200 import pa

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    wl = CONFIGS[args.config]
    K, Wm = args.steps, args.warmup
    if wl.n_steps is not None:                                                 # never run past the end of a fixed schedule
        K = max(1, min(K, wl.n_steps - Wm - 8))
    run = Runner(pa, wl, rank_seed(wl, rank), args.rng, args.couplings, dist=dist if world > 1 else None)
    pop = run.pop
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")          # > 126 MB L2
    peaks, peak_src = measured_peaks()
    fused = args.api == "anneal" and wl.n_steps is not None and not wl.multi_histogram
    sampler = ClockSampler(local) if rank == 0 else None
    t = timed_steps(torch, run, K, Wm, flush, fused, sampler, dist.barrier if world > 1 else None)
    clocks = sampler.stop() if rank == 0 else None
    obs = t["obs"]
    resample = instrumented_steps(run, min(K, 5), peaks)
    total_ms, updates_all = reduce_over_ranks(t["total_ms"], t["updates"], "cuda", dist if world > 1 else None)
    if world > 1:
        dist.barrier()
    value = updates_all / (total_ms * 1e6)

    # ---- end to end through the C ABI with HOST buffers: the population lives in pinned host memory between steps
    Ke = max(1, min(K, args.e2e_steps, run.left()))
    G = (pop.capacity + 31) // 32
    host_words = torch.empty((G, wl.N), dtype=torch.int32, pin_memory=True)
    host_E = torch.empty(pop.capacity, dtype=torch.int32, pin_memory=True)
    host_M = torch.empty(pop.capacity, dtype=torch.int32, pin_memory=True)
    pop.get_words(host_words)
    R_host = pop.population
    h2d = d2h = upd_e = 0
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    # fixed schedules: ONE C-ABI call per step with host buffers (pa_step_host: upload, resample, sweeps in chunks with the finished
    # chunks travelling back beside them, energies, observables); the adaptive workload keeps the single calls (its bisection and
    # histogram fold sit between them)
    one_call = run.betas is not None and not wl.multi_histogram
    step_s = []
    for s in range(Ke):
        ts = time.perf_counter()
        nb = ((R_host + 31) // 32) * wl.N * 4
        h2d += nb
        if one_call:
            run.i += 1
            beta = run.betas[min(run.i, len(run.betas) - 1)]
            o, _ = pop.step_host(R_host, host_words, run.beta, beta, wl.theta, host_words, host_E, host_M)
            run.beta = beta
        else:
            pop.set_words(R_host, host_words)
            o = run.step()
            pop.energies_into(host_E, host_M)
            pop.get_words(host_words)
        R_host = pop.population
        d2h += ((R_host + 31) // 32) * wl.N * 4 + 8 * R_host + ctypes.sizeof(pa.pa_obs_t)
        upd_e += o["R"] * wl.N * wl.theta
        step_s.append(time.perf_counter() - ts)                               # both step forms end synchronised with the host
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    dt, upd_e = reduce_over_ranks(dt, upd_e, "cuda", dist if world > 1 else None)
    e2e = {"value": upd_e / (dt * 1e9), "unit": UNIT, "h2d_bytes_per_step": h2d // Ke, "d2h_bytes_per_step": d2h // Ke,
           "steps": Ke, "ms_of_each_step": [round(x * 1e3, 3) for x in step_s], "what": f"{Ke} steps (capped by --e2e-steps: the packed population is {h2d // Ke / 1e9:.2f} GB each way per step): "
                                "population words pinned-host -> device, one temperature step, energies + words + observables back to host; host wall clock; "
                                + ("one pa_step_host call per step (device-to-host copies of finished chunks overlap the sweeps)" if one_call
                                   else "pa_set_words + single calls + pa_energies + pa_get_words"),
           "api": "pa_step_host" if one_call else "single calls"}
    del host_words, host_E, host_M

    # ---- weighted average of the ranks' populations at the last temperature (Eq. 6-7): the method's own exchange step
    combined = combine_over_ranks(pop.lnZ, pop.observables(run.beta), "cuda", dist if world > 1 else None, pa.pa_weighted_average)
    if rank != 0:
        run.close()
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- roofline of the dominant kernel (the sweep), live from the library's CUDA events on its stream
    roofline = roofline_of(args.rng, wl.name, t["sweep_ms"], t["sweep_updates"], t["total_ms"], peaks, peak_src)
    roofline["algorithmic_bytes_per_launch"] = 2 * ((obs["R"] + 31) // 32) * wl.N * 4
    # the integer-pipe peaks behind `peak`, re-measured live by the library's microbenchmarks (dependent chains on every SM)
    try:
        cal = {}
        for kind, name in ((0, "lop3"), (1, "imad_wide_u32"), (2, "philox_round_mix")):
            gi, mhz = pa.pa_calibrate(kind)
            cal[name + "_G_per_s"] = gi
            cal["sm_mhz"] = mhz
        cal["imad_wide_lanes_per_clk_per_sm"] = cal["imad_wide_u32_G_per_s"] * 1e3 / (cal["sm_mhz"] * n_sm())
        roofline["calibration"] = cal
        if args.rng == "philox":
            # next to the nominal peak (32 lanes/clk/SM, the strictest of the three roofs of DESIGN.md Sec. 6.1): the pipe rate the
            # library's own dependent-chain microbenchmark reaches on this GPU in this run
            roofline["peak_measured"] = cal["imad_wide_u32_G_per_s"]
            roofline["frac_measured"] = roofline["achieved"] / cal["imad_wide_u32_G_per_s"]
            roofline["peak_measured_source"] = "pa_calibrate(1): IMAD.WIDE.U32 chains on every SM, this run"
    except Exception as e:                                                    # never lose the bench line over the side measurement
        roofline["calibration"] = {"error": str(e)}
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
           "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "u32", "data": "synthetic",
           "config": {"workload": wl.name, "L": wl.L, "R_per_gpu": wl.R, "theta": wl.theta, "beta_from": wl.beta0, "rng": args.rng, "couplings": args.couplings,
                      "api": "pa_anneal, one temperature step per call" if fused else "pa_resample + pa_sweep + pa_observables per step",
                      "schedule": ("adaptive (Eq. 8), timed: steps %d-%d from beta = %g" % (Wm + 1, Wm + K, wl.beta0)
                                   + ("; rank 0 decides every step and broadcasts it (PAPER.md L118)" if world > 1 else "")) if wl.n_steps is None else
                                  f"steps {Wm + 1}-{Wm + K} of {wl.n_steps} equal steps from {wl.beta0} to {wl.beta_f} are the timed ones "
                                  f"(beta <= {wl.betas()[min(Wm + K, wl.n_steps)]:.4g}); the whole schedule: --whole-run",
                      "l2": "flushed between timed steps (256 MiB memset outside the CUDA events)",
                      "parallelism": "independent populations per GPU" if world > 1 else "1 GPU"},
           "clocks": clocks, "e2e": e2e, "gpu_launches": t["launches"], "roofline": roofline, "resample": resample,
           "last_observables": obs, "combined_observables": combined}
    if world == 1 and args.couplings == "ferro" and (args.whole_run or (args.whole_run is None and args.config <= 4)):
        out["whole_run"] = whole_run(pa, wl, rank_seed(wl, rank), args.rng)
    run.close()
    del run, pop
    torch.cuda.empty_cache()
    if world == 1 and not args.no_others and args.couplings == "ferro":
        # configs 1-2 are launch/latency-bound and the roofline is judged on the large ones; all stay visible here
        others = []
        for cfg, rng in [(c, args.rng) for c in (2, 3, 4) if c != args.config] + [(5, "lcg"), (3, "lcg"), (6, "philox")]:
            if (cfg, rng) == (args.config, args.rng):
                continue
            try:
                others.append(sub_record(torch, pa, cfg, rng, flush, peaks, peak_src))
            except Exception as e:                                            # a side record never costs the bench line
                others.append({"workload": CONFIGS[cfg].name, "rng": rng, "error": repr(e)})
        out["other_configs"] = others
    out["cpu_baseline"] = cpu_baseline(wl, args.rng) if world == 1 and not args.no_cpu and args.couplings == "ferro" else None
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def oracle_step_rate(wl, R_sample, steps, warmup, rng="philox"):
    """The oracle, as it stands, on a population of R_sample replicas of the workload's shape."""
    from oracle import pa_oracle as po
    o = po.Oracle(wl.L, R_sample, wl.seed, dims=wl.dims)
    if rng == "lcg":
        o.set_rng_mode(po.RNG_LCG)
    betas = wl.betas() if wl.n_steps is not None else [wl.beta0 + 0.005 * i for i in range(steps + warmup + 2)]
    i, beta_prev = 0, betas[0]
    for _ in range(warmup):
        i += 1
        o.resample(beta_prev, betas[i]); o.sweep(betas[i], wl.theta); o.observables(betas[i]); beta_prev = betas[i]
    upd, t0 = 0, time.perf_counter()
    for _ in range(steps):
        i += 1
        o.resample(beta_prev, betas[i]); o.sweep(betas[i], wl.theta); ob = o.observables(betas[i]); beta_prev = betas[i]
        upd += ob["R"] * wl.N * wl.theta
    dt = time.perf_counter() - t0
    return upd / (dt * 1e9), dt / steps * 1e3, po.num_threads()


def oracle_step_rates(wl, R_sample, steps, rng="philox"):
    """updates/ns of each of `steps` consecutive temperature steps of the oracle on R_sample replicas, and the thread count."""
    from oracle import pa_oracle as po
    o = po.Oracle(wl.L, R_sample, wl.seed, dims=wl.dims)
    if rng == "lcg":
        o.set_rng_mode(po.RNG_LCG)
    betas = wl.betas() if wl.n_steps is not None else [wl.beta0 + 0.002 * i for i in range(steps + 2)]
    out = []
    for i in range(1, steps + 1):
        t0 = time.perf_counter()
        o.resample(betas[i - 1], betas[i]); o.sweep(betas[i], wl.theta); ob = o.observables(betas[i])
        out.append(ob["R"] * wl.N * wl.theta / ((time.perf_counter() - t0) * 1e9))
    return out, po.num_threads()


def cpu_baseline(wl, rng="philox"):
    """The oracle as it stands on the host cores: one warm-up step (first-touch page faults, OpenMP start-up), then the median of
    three timed steps, on the slice SURVEY 8(d) prescribes (the full population for configs 1-3, 4096 replicas for configs 4-5,
    capped at ~3e9 spin updates per step); and on one thread (the paper's CPU figure, Table 2: 22.5-23.1 ns per update = 0.044
    updates/ns on one Xeon core) on an eighth of that slice, one warm-up + two timed steps."""
    from oracle import pa_oracle as po
    R_s = min(wl.R, 4096 if wl.R * wl.N > 10**9 else wl.R, max(256, int(3.0e9 / (wl.N * wl.theta))))
    R_1 = max(32, R_s // 8)

    def rates(R, steps):
        out, cores = [], None
        o_steps = steps + 1
        per = oracle_step_rates(wl, R, o_steps, rng)
        cores = per[1]
        out = sorted(per[0][1:])                                                # drop the warm-up step
        return out[len(out) // 2], cores

    v, cores = rates(R_s, 3)
    po.set_num_threads(1)
    v1, _ = rates(R_1, 2)
    po.set_num_threads(cores)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "ms_per_step": R_s * wl.N * wl.theta / (v * 1e6),
            "value_one_thread": v1, "timed_steps": 3, "warmup_steps": 1,
            "sample": f"median of 3 temperature steps (resample + {wl.theta} sweeps + observables) after 1 warm-up step, R={R_s} replicas of "
                      f"{wl.name} (L={wl.L}), oracle/pa_oracle.cpp -O2 OpenMP on {cores} threads; one thread: R={R_1}, 2 timed steps"}


def run_reference(args):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    wl = CONFIGS[args.config]
    R_s = min(wl.R, max(256, int(2.0e8 / (wl.N * wl.theta))))               # bounded sample per step
    v, ms, cores = oracle_step_rate(wl, R_s, args.steps, args.warmup, args.rng)
    sample = f"each step = one temperature step of R={R_s} replicas of {wl.name} (L={wl.L}, theta={wl.theta}); CPU oracle, OpenMP"
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "u8", "data": "synthetic",
           "config": {"workload": wl.name, "L": wl.L, "R_per_gpu": wl.R, "theta": wl.theta, "sample_R": R_s},
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, choices=sorted(CONFIGS),
                    help="BASELINE.json configs index + 1; default 5 = the largest single-GPU configuration (L=256, R=10^6)")
    ap.add_argument("--e2e-steps", type=int, default=2, help="steps of the host-buffer end-to-end leg (cfg5 moves 8.2 GB each way per step)")
    ap.add_argument("--no-others", action="store_true", help="skip the compact records of the other configurations / the LCG stream")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--whole-run", dest="whole_run", action="store_true", default=None,
                    help="also time the config's whole schedule (t_SF, Eq. 11); default: on for configs 1-4 (seconds), off for 5 (minutes)")
    ap.add_argument("--api", default="steps", choices=["steps", "anneal"],
                    help="timed steps through the single calls (default) or through pa_anneal, one step per call (fixed schedules)")
    ap.add_argument("--couplings", default="ferro", choices=["ferro", "pmj"],
                    help="ferromagnet (default, Eq. 10) or a seeded random +-J sample (second workload, PAPER.md L313; context)")
    ap.add_argument("--theta-scan", action="store_true", help="re-measure the paper's Table 3 / Table 4 theta dependence (context)")
    ap.add_argument("--no-whole-run", dest="whole_run", action="store_false")
    ap.add_argument("--rng", default="philox", choices=["philox", "lcg"],
                    help="sweep stream: one Philox number per spin (default, O1) or the paper's Philox-seeded LCG (O11, L236-L241)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.theta_scan:
        theta_scan(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
