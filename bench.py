#!/usr/bin/env python
"""bench.py — whole hot path (im_reset + im_rollout + im_returns) on synthetic BASELINE.json configs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

One "step" = one pass of the whole hot path over one batch: reset to empty pools, T-tick rollout of all E
envs under the random policy (decision logs on), then GAE + Lagrangian returns.
Prints ONE JSON line (contract in the task statement).  Default workload: configs[4] (the largest, the "full
training-step workload"); `--config 1..5` selects another.  N > 1 (torchrun): every rank runs the full config on
its own env-id range (weak scaling, no data-path collective; one all-reduce of the four scalars behind
C-bar / U-bar / sigma_U per step).
"""
from __future__ import annotations

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

from im_workload import CONFIGS, make_policy_blob, make_pool_spec  # noqa: E402

DEFAULT_CONFIG = 5
GAMMA, LAM, MU = 0.99, 0.95, 0.5


def csrc_sha():
    """First 12 hex digits of the sha256 over the kernel sources (name-sorted): ties an ncu capture to the code it profiled."""
    import hashlib
    d = os.path.join(ROOT, "paper_2606_11440_b200", "csrc")
    h = hashlib.sha256()
    for name in sorted(os.listdir(d)):
        h.update(name.encode()); h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:12]


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=float(d["hbm_gbs"]), bf16_burst=float(d["bf16_tflops"]), bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), src="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, src="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._pump, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t_begin, t_end):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        for ts, line in self.rows:
            if ts < t_begin - 0.05 or ts > t_end + 0.15:
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            for ts, line in self.rows[-3:]:
                f = [x.strip() for x in line.split(",")]
                try:
                    sm.append(float(f[0])); mx = float(f[1])
                except Exception:
                    pass
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=mx, reasons=sorted(reasons), samples=len(sm))


def algorithmic_model(spec, counters_sum, T, E):
    """Algorithmic bytes / flops of one step from the run's own counters."""
    N = spec.n_models
    n_run, n_wait = float(counters_sum[12]), float(counters_sum[13])
    n_exec, n_arr = float(counters_sum[11]), float(counters_sum[0])
    env_ticks = float(E) * T
    serve_bytes = 8 * n_run                                     # k_serve: the slots of the running requests, read + write
    sim_bytes = 4 * n_wait + (24 * N + 10) * env_ticks + 52 * n_exec + 16 * n_arr   # k_sim: everything else of SURVEY 8(d)
    F, H = spec.f_in, spec.hidden
    mac_exec = F * H + H * H + H * (3 * N + 1)
    mac_plan = F * H + H * H + H * 24
    exec_flops = 2.0 * mac_exec * (n_exec + env_ticks + E)      # decisions + one critic row per env-tick (+ bootstrap row)
    plan_flops = 2.0 * mac_plan * float(counters_sum[10])
    exec_bytes = (24 + 4) * n_exec + (12 * N + 4) * (env_ticks + E)   # row r/w + snapshot read + val write
    plan_bytes = (20 + 24) * float(counters_sum[10])
    # returns: GAE reads 13 B and writes 8 B per env-tick; the utility pass reads a 16-byte query record, the
    # normalisation pass reads it again and writes 4 B (R32)
    ret_bytes = 21.0 * env_ticks + 36.0 * float(counters_sum[2])
    return dict(sim_bytes=sim_bytes, serve_bytes=serve_bytes, exec_flops=exec_flops, plan_flops=plan_flops, exec_bytes=exec_bytes, plan_bytes=plan_bytes,
                ret_bytes=ret_bytes, n_exec=n_exec, n_plan=float(counters_sum[10]), env_ticks=env_ticks)


def sim_access_model(spec, counters_sum, T, E):
    """What one k_sim launch has to move, per launch (= E env-ticks), split by how the memory system sees it
    (DESIGN.md section 7 'what bounds k_sim'): `stream_*` sectors are read / written in lane order by whole warps or by
    the bulk copies (header in + out, k_serve's results, issue records, snapshot, trajectory rows); `rand_*` are the
    ALGORITHMIC accesses at data-dependent addresses that no layout of per-request records can avoid: per admission a
    full 32-byte slot record and the slot's token counter (a 2-byte store into a sector: fill + write), per completion
    the slot record and the query entry read and the query's plan word written back, per arrival the query entry."""
    N = spec.n_models
    SP = int(sum(((int(x) + 7) // 8) * 8 for x in spec.slots))
    n_chunks = spec.rcap // 32 + N
    hdr_words = 3 * N + (SP + 31) // 32 + 2 + spec.qcap // 32 + (n_chunks + 3) // 4 + 4 + 2      # im_api.cu: carve()
    cm_words = (SP // 8 + 3) // 4
    per_tick = 1.0 / T
    n_exec, n_arr, n_done, n_fin = (float(counters_sum[i]) * per_tick for i in (11, 0, 6, 2))
    stream_read = E * (hdr_words + cm_words + N) * 4 / 32.0 + n_exec * 8 / 32.0
    stream_write = E * (hdr_words * 4 + 12 * N + 10) / 32.0 + (n_exec + n_arr + n_fin) * 16 / 32.0   # + rows / log records
    rand = dict(read16=2.0 * n_done, write32=n_exec, write16=n_exec + (n_done - n_fin) + n_arr)
    return dict(stream_read_sectors=stream_read, stream_write_sectors=stream_write, rand_ops=rand, hdr_words=hdr_words)


def random_access_report(spec, csum, T, E, cfg, dev, peaks, sim_ms):
    """roofline['random_access']: measured rates of the device for accesses at data-dependent addresses, and two lower
    bounds of one k_sim launch built from them: `t_alg_ms` from the algorithmic access counts of `sim_access_model`,
    `t_traffic_ms` from the DRAM sectors ncu counted for that launch (profiles/ncu_sim_dram.csv, used only while the
    kernel sources still hash to the capture's)."""
    from paper_2606_11440_b200.probe import random_access_rates
    rates = random_access_rates(device=str(dev), gib=16)
    m = sim_access_model(spec, csum, T, E)
    hbm = peaks["hbm"] * 1e9
    t_stream = (m["stream_read_sectors"] + m["stream_write_sectors"]) * 32.0 / hbm
    t_alg = t_stream + sum(m["rand_ops"][k] / (rates[k] * 1e9) for k in m["rand_ops"])
    out = {"peak_gops": rates, "peak_source": "libimprobe (include/im_probe.h), 1 MiB windows, measured in this run",
           "alg_ops_per_launch": m["rand_ops"], "stream_sectors_per_launch": m["stream_read_sectors"] + m["stream_write_sectors"],
           "t_alg_ms": t_alg * 1e3, "frac_alg": t_alg * 1e3 / max(sim_ms, 1e-9), "t_traffic_ms": None, "frac_traffic": None}
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "ncu_sim_dram.csv")) as f:
            for row in csv.DictReader(f):
                if row["config"] == f"cfg{cfg}" and E == CONFIGS[cfg]["E"] and row["csrc_sha"] == csrc_sha():
                    rd, wr = float(row["dram_sectors_read"]), float(row["dram_sectors_write"])
                    r_rand, w_rand = max(rd - m["stream_read_sectors"], 0.0), max(wr - m["stream_write_sectors"], 0.0)
                    t_tr = t_stream + r_rand / (rates["read16"] * 1e9) + w_rand / (rates["write32"] * 1e9)
                    out.update(dram_sectors_per_launch={"read": rd, "write": wr}, t_traffic_ms=t_tr * 1e3, frac_traffic=t_tr * 1e3 / max(sim_ms, 1e-9))
    except (OSError, ValueError, KeyError):
        pass
    return out


def baseline_sample(cfg: int, cores: int):
    """(envs, ticks) of the bounded sample the oracle is timed on: the first envs x the first ticks of the config."""
    return max(cores * 4, 32), {1: 200, 2: 500, 3: 300, 4: 200, 5: 512}[cfg]


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle, as it stands, on the box's host cores, on a bounded sample of the workload."""
    if rank != 0:
        return
    from oracle import oracle as O
    cfg = args.config
    full = CONFIGS[cfg]
    cores = os.cpu_count() or 1
    n_envs, T = baseline_sample(cfg, cores)              # the same sample as the cpu_baseline leg of the main arm
    spec = make_pool_spec(cfg, n_envs=n_envs, n_ticks=T)
    blob = make_policy_blob(spec)
    o = O.Oracle(spec, seed=0)
    times, decs = [], 0
    for i in range(args.warmup + args.steps):
        o.reset()
        t0 = time.perf_counter()
        o.rollout(blob, T, n_threads=cores)
        o.returns(GAMMA, LAM, MU)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
            decs += int(o.counters()[:, 11].sum())
    tot = sum(times)
    val = n_envs * T * len(times) / tot
    sample = f"first {n_envs} of {full['E']} envs x {T} of {full['T']} ticks per step (envs are independent)"
    line = {"impl": "reference", "metric": "env_ticks_per_sec", "value": val, "unit": "env-ticks/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if spec.policy_dtype == 0 else "bf16", "data": "synthetic",
            "config": {"workload": f"configs[{cfg - 1}] (sampled)", "E": n_envs, "T": T, "n_models": spec.n_models},
            "agent_decisions_per_sec": decs / tot,
            "cpu_baseline": {"value": val, "unit": "env-ticks/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "env-ticks/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def cpu_baseline(cfg: int, budget_s: float = 15.0):
    """The oracle timed on the host cores on a bounded sample of the same workload (about 10-30 s of CPU work)."""
    from oracle import oracle as O
    cores = os.cpu_count() or 1
    n_envs, T = baseline_sample(cfg, cores)
    full = CONFIGS[cfg]
    spec = make_pool_spec(cfg, n_envs=n_envs, n_ticks=T)
    blob = make_policy_blob(spec)
    o = O.Oracle(spec, seed=0)
    o.rollout(blob, min(T, 8), n_threads=cores)     # page in
    o.reset()
    t0 = time.perf_counter()
    reps = 0
    while True:
        o.reset()
        o.rollout(blob, T, n_threads=cores)
        o.returns(GAMMA, LAM, MU)
        reps += 1
        el = time.perf_counter() - t0
        if el > budget_s:
            break
    return {"value": n_envs * T * reps / el, "unit": "env-ticks/s", "cores": cores, "kind": "oracle",
            "sample": f"{reps} x (first {n_envs} of {full['E']} envs x first {T} of {full['T']} ticks), {el:.1f} s, OpenMP over envs"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--envs", type=int, default=None, help="override E (debug)")
    ap.add_argument("--ticks", type=int, default=None, help="override T (debug)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-probe", action="store_true", help="skip the random-access probe (libimprobe)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2606_11440_b200 import (InfraMind, IM_TEL_ADV, IM_TEL_RET, IM_TEL_SCALARS, build)
    from paper_2606_11440_b200.sharding import allreduce_sums
    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    cfg = args.config
    spec = make_pool_spec(cfg, n_envs=args.envs, n_ticks=args.ticks)
    E, T = spec.n_envs, spec.n_ticks
    spec = spec.with_(env_id_base=rank * E)          # weak scaling: each rank owns its own env-id range
    blob_host = make_policy_blob(spec, seed=0)
    blob_dev = torch.from_numpy(blob_host).to(dev)
    seeds = [0, 1, 2, 3, 4] if cfg == 5 else [0]     # configs[4]: "Seeds 0-4"
    stream = torch.cuda.Stream(device=dev)
    ctxs, arena = [], None
    with torch.cuda.stream(stream):
        for s in seeds:
            c = InfraMind(spec, seed=s, device=dev, debug_flags=1, stream=stream, arena=arena)
            arena = c.arena
            ctxs.append(c)
    peaks = _peaks()

    chunk = spec.max_ticks                           # configs 3-4: 4000 ticks = 8 x im_rollout(500), state persists

    def step(i, blob):
        c = ctxs[i % len(ctxs)]
        c.reset()
        done = 0
        while done < T:
            n = min(chunk, T - done)
            c.rollout(blob, n)
            c.returns(GAMMA, LAM, MU)
            if world > 1:
                # the step's one collective: the four sums behind C-bar / U-bar / sigma_U over all ranks;
                # every rank then re-normalises its UNORM with the job's statistics inside the library
                c.returns_finish(allreduce_sums(c.sums(), device=dev))
            done += n
        return c

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: inputs (weights, tables) already in HBM
    for i in range(args.warmup):
        step(i, blob_dev)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = sum(c.launches for c in ctxs)
    barrier()
    t_begin = time.time()
    ev0.record(stream)
    for i in range(args.steps):
        step(args.warmup + i, blob_dev)
    ev1.record(stream)
    barrier()
    t_end = time.time()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop(t_begin, t_end)
    launches = sum(c.launches for c in ctxs) - launches0
    last = ctxs[(args.warmup + args.steps - 1) % len(ctxs)]
    csum = last.counters().sum(axis=0)
    sc = last.scalars()
    if world > 1:
        tms = torch.tensor([ms], device=dev, dtype=torch.float64)
        dist.all_reduce(tms, op=dist.ReduceOp.MAX)
        ms = float(tms.item())
    ms_per_step = ms / args.steps
    env_ticks_per_s = world * E * T / (ms_per_step * 1e-3)
    model = algorithmic_model(spec, csum, T, E)
    decisions_per_s = world * model["n_exec"] / (ms_per_step * 1e-3)

    # ---- per-kernel-class device times (CUDA events inside the library, same launches) for the roofline
    for c in ctxs:
        c.set_profiling(True)
    ksteps = max(1, min(args.steps, 2))
    for i in range(ksteps):
        cprof = step(args.warmup + args.steps + i, blob_dev)
    kt = {"sim": [0.0, 0], "plan": [0.0, 0], "exec": [0.0, 0], "returns": [0.0, 0], "serve": [0.0, 0]}
    for c in ctxs:
        for k, (m, n) in c.kernel_times().items():
            kt[k][0] += m; kt[k][1] += n
        c.set_profiling(False)
    tot_k = sum(v[0] for v in kt.values()) or 1.0
    share = {k: v[0] / tot_k for k, v in kt.items()}
    dominant = max(("sim", "serve", "plan", "exec"), key=lambda k: kt[k][0])
    per_launch_ms = {k: (v[0] / v[1] if v[1] else 0.0) for k, v in kt.items()}
    n_l = {k: (kt[k][1] / ksteps if kt[k][1] else 1.0) for k in kt}      # launches (timed brackets) of the class per step
    bf16 = spec.policy_dtype == 1
    tunit = "GB per launch (ncu dram__bytes_read+write)"
    if dominant in ("sim", "serve"):
        achieved = model[dominant + "_bytes"] / n_l[dominant] / (per_launch_ms[dominant] * 1e-3) / 1e9
        roof = {"bound": "hbm", "kernel": "k_" + dominant, "achieved": achieved, "peak": peaks["hbm"], "unit": "GB/s",
                "frac": achieved / peaks["hbm"], "traffic": None, "traffic_unit": tunit}
    else:
        fl = model["exec_flops"] if dominant == "exec" else model["plan_flops"]
        achieved = fl / n_l[dominant] / (per_launch_ms[dominant] * 1e-3) / 1e12
        if bf16:
            pk = peaks["bf16_sustained"]
            kname = "k_policy_tc" + f"<{dominant}>"
            roof = {"bound": "tensor", "kernel": kname, "achieved": achieved, "peak": pk, "unit": "TFLOP/s", "frac": achieved / pk, "traffic": None, "traffic_unit": tunit}
        else:
            pk = 148 * 128 * 2 * 1.965e9 / 1e12       # fp32 FFMA: 148 SMs x 128 lanes x 2 flop x max clock
            roof = {"bound": "alu", "kernel": f"k_policy_f32<{dominant}>", "achieved": achieved, "peak": pk, "unit": "TFLOP/s", "frac": achieved / pk, "traffic": None, "traffic_unit": tunit}
    # DRAM bytes per launch of the dominant kernel: taken from the committed ncu --set full capture only if that capture was
    # made from the kernel sources this run was built from (sha256 of csrc/, first 12 hex digits); otherwise null
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if (row["config"] == f"cfg{cfg}" and row["kernel"] == roof["kernel"] and E == CONFIGS[cfg]["E"]
                        and row["csrc_sha"] == csrc_sha()):
                    roof["traffic"] = float(row["dram_bytes_per_launch"]) / 1e9
                    roof["traffic_source"] = row["source"]
    except (OSError, ValueError, KeyError):
        pass
    roof["csrc_sha"] = csrc_sha()
    roof["peak_source"] = f"MEASURED_PEAKS.json ({peaks['src']})"
    roof["kernel_share_of_step"] = share
    roof["kernel_ms_per_launch"] = per_launch_ms
    per_s = lambda key, cls: model[key] / n_l[cls] / max(per_launch_ms[cls] * 1e-3, 1e-12)
    roof["sim_hbm_frac"] = per_s("sim_bytes", "sim") / 1e9 / peaks["hbm"]
    roof["serve_hbm_frac"] = per_s("serve_bytes", "serve") / 1e9 / peaks["hbm"]
    # the tick simulation as a whole (k_serve + k_sim: the SURVEY 8(d) byte formula over both kernels' time)
    t_tick = per_launch_ms["sim"] * n_l["sim"] + per_launch_ms["serve"] * n_l["serve"]
    roof["tick_sim_hbm_frac"] = (model["sim_bytes"] + model["serve_bytes"]) / max(t_tick * 1e-3, 1e-12) / 1e9 / peaks["hbm"]
    roof["exec_tensor_frac"] = per_s("exec_flops", "exec") / 1e12 / peaks["bf16_sustained"] if bf16 else None
    roof["plan_tensor_frac"] = per_s("plan_flops", "plan") / 1e12 / peaks["bf16_sustained"] if bf16 else None
    roof["step_hbm_frac"] = (model["sim_bytes"] + model["serve_bytes"] + model["exec_bytes"] + model["plan_bytes"] + model["ret_bytes"]) / (ms_per_step * 1e-3) / 1e9 / peaks["hbm"]
    roof["step_tensor_frac"] = (model["exec_flops"] + model["plan_flops"]) / (ms_per_step * 1e-3) / 1e12 / peaks["bf16_sustained"] if bf16 else None
    # t_lb / t, t_lb = the larger of the two bound times of the whole step
    roof["step_lb_frac"] = max(roof["step_hbm_frac"], roof["step_tensor_frac"] or 0.0)
    # one im_returns call covers one rollout call (chunk): bytes of that call over the time of that call
    roof["returns_hbm_frac"] = per_s("ret_bytes", "returns") / 1e9 / peaks["hbm"]
    # ---- k_sim against the ceilings that apply to it: accesses at data-dependent addresses (libimprobe, measured now)
    if rank == 0 and not args.no_probe:
        try:
            roof["random_access"] = random_access_report(spec, csum, T, E, cfg, dev, peaks, per_launch_ms["sim"])
        except Exception as err:  # the probe is a measurement aid: never fail the bench line over it
            roof["random_access"] = {"error": str(err)[:200]}

    # ---- end to end through the C ABI with HOST buffers: host blob in, ADV / RET / scalars out to pinned host memory
    adv_h = torch.empty((chunk, E), dtype=torch.float32, pin_memory=True)
    ret_h = torch.empty((chunk, E), dtype=torch.float32, pin_memory=True)
    e2e_steps = max(1, min(args.steps, 2))
    step(0, blob_host)
    barrier()
    ee0, ee1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ee0.record(stream)
    d2h = 0
    for i in range(e2e_steps):
        c = ctxs[(i + 1) % len(ctxs)]
        c.reset()
        done, d2h = 0, 0
        while done < T:
            n = min(chunk, T - done)
            c.rollout(blob_host, n)
            c.returns(GAMMA, LAM, MU)
            d2h += c.read_into(IM_TEL_ADV, adv_h) + c.read_into(IM_TEL_RET, ret_h) + 64
            c.scalars()
            done += n
    ee1.record(stream)
    barrier()
    e2e_ms = ee0.elapsed_time(ee1) / e2e_steps
    if world > 1:
        tms = torch.tensor([e2e_ms], device=dev, dtype=torch.float64)
        dist.all_reduce(tms, op=dist.ReduceOp.MAX)
        e2e_ms = float(tms.item())

    if rank == 0:
        line = {
            "metric": "env_ticks_per_sec", "value": env_ticks_per_s, "unit": "env-ticks/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16" if bf16 else "f32", "data": "synthetic",
            "config": {"workload": f"configs[{cfg - 1}]: E={E} envs/GPU, {spec.n_models}-model pool, {T}-tick rollout + GAE/Lagrangian returns, "
                                   f"{'bf16' if bf16 else 'fp32'} {spec.f_in}->{spec.hidden}x2 policy, seeds {seeds}",
                       "E": E, "T": T, "n_models": spec.n_models, "qcap": spec.qcap, "rcap": spec.rcap,
                       "l2_policy": "state working set (%.1f GB) >> 126 MB L2; no flush needed" % (last.arena_bytes / 1e9),
                       "arena_gb": last.arena_bytes / 1e9},
            "agent_decisions_per_sec": decisions_per_s,
            "planner_decisions_per_sec": world * model["n_plan"] / (ms_per_step * 1e-3),
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": world * E * T / (e2e_ms * 1e-3), "unit": "env-ticks/s", "h2d_bytes_per_step": int(blob_host.nbytes) * ((T + chunk - 1) // chunk),
                    "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms},
            "roofline": roof,
            "scalars": {k: (float(v) if not isinstance(v, int) else v) for k, v in sc.items()},
        }
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(cfg)
        elif world > 1:
            line["cpu_baseline"] = None
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
