#!/usr/bin/env python
"""bench.py -- the hot path of arxiv/paper_2606_22327 on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A STEP is one pass of the whole hot path (keys -> pack -> per-instance radix sort -> admission /
feasibility -> state advance -> reductions) over one synthetic batch: one
`svf_simulate_policies` call = the simulator under all four policies (SVF, 1-bit SVF, SJF, FCFS) on
BASELINE.json configs[2] (4,096 instances x 1,000 requests, Poisson rate 4, M = 300,000), every
output requested.
metric = simulated request-steps per second, request_steps = sum_i o_i per policy run.
Per rank the batch is fixed (weak scaling); ranks hold different seeded batches; no collective
on the data path (instances are independent).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_22327_b200 import sharding as S  # noqa: E402
from paper_2606_22327_b200 import traces as T  # noqa: E402

METRIC = "simulated_request_steps_per_sec"
UNIT = "request-steps/s"
POLICIES = (0, 1, 2, 3)
POLICY_NAMES = ("svf", "svf_1bit", "sjf", "fcfs")
L2_FLUSH_BYTES = 512 << 20

# The dominant kernel (k_sim_slots, phase B) is bound by integer ALU issue, not by HBM (its state
# is on chip).  Algorithmic work per launch = 4*E + 2*U lane-operations: E = running
# entries examined over all head evaluations (two compares, one add, one max each), U = running
# entries updated over all admissions (one compare, one add each); both counted exactly by the
# kernel's counting variant on the same inputs.  Peak = the SM issue rate, from the guide's unit
# counts: SMs x 4 schedulers x 32 lanes x 1 warp-instruction/cycle x max SM clock.
OPS_PER_EXAMINED, OPS_PER_UPDATED = 4, 2
# HBM bytes per request and policy the same kernel must move: a, s, o (12) + rank (4) +
# start, finish (8) + latency for the p99 selection (4 written, 4 read back); the register-queue
# kernels write their outputs in index order and never read order[]
SIM_BYTES_PER_REQUEST = 32
# dram__bytes_read.sum + dram__bytes_write.sum of one k_sim_slots launch on this workload come from the
# committed `ncu --set full` summary of the same command (never from a run under the profiler here)
SIM_PROFILE = os.path.join("profiles", "r03_kslots_traffic.json")


def _sources_sha256(files):
    import hashlib
    h = hashlib.sha256()
    for f in files:
        h.update(open(os.path.join(ROOT, f), "rb").read())
    return h.hexdigest()


def profiled_dram_traffic():
    """(bytes per k_sim_slots launch, source) from the small JSON that sits beside the committed
    `ncu --set full` summary and names its table, or (None, why) -- also when the simulator sources are
    no longer the ones that were profiled (their SHA-256 is stamped in the file)."""
    path = os.path.join(ROOT, SIM_PROFILE)
    try:
        rec = json.load(open(path))
        total = float(rec["dram__bytes_read.sum"]) + float(rec["dram__bytes_write.sum"])
        if _sources_sha256(rec["source_files"]) != rec["source_sha256"]:
            return None, f"{SIM_PROFILE} was captured from other simulator sources (commit {rec.get('commit', '?')}): capture again"
        return total, f"{SIM_PROFILE}: {rec.get('table', '?')} (sources as of commit {rec.get('commit', '?')})"
    except (OSError, KeyError, ValueError):
        return None, f"{SIM_PROFILE} missing or unreadable"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--instances", type=int, default=4096)
    ap.add_argument("--requests", type=int, default=1000)
    ap.add_argument("--lam", type=float, default=4.0)
    ap.add_argument("--e2e-chunks", type=int, default=8, help="instance chunks (streams) of the end-to-end leg")
    ap.add_argument("--no-extras", action="store_true", help="skip the per-kernel and per-config extras")
    ap.add_argument("--extras-file", default=None, help=f"where the extras go (default {EXTRAS_FILE}); never stdout")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-oracle-extras", action="store_true", help="extras without the oracle timed beside each config")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def alu_peak(torch, dev):
    """Issue-rate roofline in lane-operations/s: SMs x 4 schedulers x 32 lanes x max SM clock."""
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    mhz, src = 1965.0, "B200_PROFILING.md max SM clock 1965 MHz"
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            mhz, src = float(json.load(open(p))["sm_max_mhz"]), "MEASURED_PEAKS.json sm_max_mhz"
        except Exception:
            pass
    return sms * 4 * 32 * mhz * 1e6, f"{sms} SMs x 4 schedulers x 32 lanes x {mhz:g} MHz ({src})"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ts, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                c, m = float(f[0]), float(f[1])
            except ValueError:
                continue
            if t0 - 0.05 <= ts <= t1 + 0.15:
                sm.append(c); mx.append(m)
                for nm, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
        if not sm:   # region shorter than one sample: take whatever we saw
            for ts, line in self.rows:
                f = [x.strip() for x in line.split(",")]
                try:
                    sm.append(float(f[0])); mx.append(float(f[1]))
                except Exception:
                    pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def make_batch(args, rank):
    lo, hi = S.weak_shard(rank, args.instances)        # per-GPU work fixed: weak scaling
    return T.config3(n_instances=hi - lo, n=args.requests, lam=args.lam, first_instance=lo)


# ---------------------------------------------------------------------------------------------
# reference arm = the CPU oracle, as it stands, on the host cores (tier framing (4))
# ---------------------------------------------------------------------------------------------
def oracle_step(svf_ref, sample, threads):
    dec = 0
    for p in POLICIES:
        r = svf_ref.simulate(sample, p, n_threads=threads)
        dec += int(r.decisions.sum())
    return dec


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import svf_ref
    svf_ref.build()
    threads = min(os.cpu_count() or 1, svf_ref.max_threads())
    n_inst = args.instances                        # the same batch as the repo arm's rank 0 (about 1.5 s per step on 16 cores)
    sample = T.config3(n_instances=n_inst, n=args.requests, lam=args.lam)
    rs = sample.request_steps * len(POLICIES)
    for _ in range(max(args.warmup, 0) and 1):
        oracle_step(svf_ref, sample, threads)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(svf_ref, sample, threads)
    dt = time.perf_counter() - t0
    val = rs * args.steps / dt
    desc = (f"all {n_inst} instances x {args.requests} requests x 4 policies per step, instance-parallel over {threads} "
            f"host threads (nproc {os.cpu_count()})")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64",
            "data": "synthetic", "config": workload_config(args, n_inst),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(args, n_inst=None):
    return {"workload": "BASELINE.json configs[2] batched simulation: "
                        f"{n_inst or args.instances} instances x {args.requests} requests, Poisson rate "
                        f"{args.lam:g}/step, lognormal s (mean 600, sigma 0.8, [16,4096]) and o (mean 250, sigma 1.0, "
                        "[1,2048]), M=300000, policies svf+svf_1bit+sjf+fcfs per step, all outputs",
            "instances_per_gpu": n_inst or args.instances, "requests_per_instance": args.requests,
            "M": 300000, "policies": list(POLICY_NAMES),
            "cache": f"L2 flushed between timed steps (write of {L2_FLUSH_BYTES >> 20} MiB)"}


# ---------------------------------------------------------------------------------------------
# the ONE line the driver reads: compact (<= HEADLINE_MAX_BYTES), strict JSON, printed before any
# extra is run; everything else goes to EXTRAS_FILE
# ---------------------------------------------------------------------------------------------
HEADLINE_MAX_BYTES = 4096
EXTRAS_FILE = os.path.join("gpurun_out", "bench_extras.json")
HEADLINE_KEYS = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                 "scaling", "vs_baseline", "dtype", "data", "config", "decisions_per_sec", "clocks", "e2e",
                 "gpu_launches", "roofline", "cpu_baseline")
ROOFLINE_KEYS = ("kernel", "bound", "achieved", "peak", "unit", "frac", "traffic", "kernel_ms", "share_of_step",
                 "algorithmic_ops_per_launch", "hbm_frac")


def _sig(x, digits=7):
    """floats to `digits` significant figures (the line is read by a program, then by people)"""
    if isinstance(x, float):
        return float(f"{x:.{digits}g}") if x == x and abs(x) != float("inf") else None
    if isinstance(x, dict):
        return {k: _sig(v, digits) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_sig(v, digits) for v in x]
    return x


def build_headline(full: dict, extras_file=None) -> str:
    """The compact headline of `full` (run_ours's whole record) as one line of strict JSON of at most
    HEADLINE_MAX_BYTES: the contract's keys, the scalar fields of `roofline`, `cpu_baseline`, `e2e`.
    Raises if a required key is missing or the line is too long (a test builds it from canned numbers)."""
    head = {k: full[k] for k in HEADLINE_KEYS if k in full}
    missing = [k for k in HEADLINE_KEYS if k not in head and k != "cpu_baseline"]
    if missing:
        raise KeyError(f"bench headline lacks {missing}")
    roof = full["roofline"]
    head["roofline"] = {k: roof.get(k) for k in ROOFLINE_KEYS}
    if isinstance(roof.get("share_of_step"), dict):      # the dominant kernel's share only
        head["roofline"]["share_of_step"] = roof["share_of_step"].get("phase_b_simulator")
    if isinstance(roof.get("hbm"), dict):
        head["roofline"]["hbm_frac"] = roof["hbm"].get("frac")
    for k in ("fingerprint_fnv1a64",):
        if k in full:
            head[k] = full[k]
    if extras_file:
        head["extras_file"] = extras_file
    text = json.dumps(_sig(_finite(head)), allow_nan=False, separators=(",", ":"))
    if len(text.encode()) > HEADLINE_MAX_BYTES:
        raise ValueError(f"bench headline is {len(text.encode())} bytes (> {HEADLINE_MAX_BYTES})")
    return text


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2606_22327_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the library has no CPU path)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    B.lib()

    batch = make_batch(args, rank)
    rs_step = batch.request_steps * len(POLICIES)
    dt_dev = B.DeviceTrace.from_host(batch, device=dev)
    outs = [B.SimOut.alloc(dt_dev) for _ in POLICIES]
    ws = torch.empty(B.svf_simulate_policies_workspace_bytes(dt_dev, len(POLICIES)), dtype=torch.uint8, device=dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def step(profile=None):
        # one call: presort under each policy, then ONE persistent launch over 4 x I work items
        B.svf_simulate_policies(dt_dev, POLICIES, outs=outs, ws=ws)
        if profile is not None:
            profile.append(B.simulate_phase_ms())
        return B.last_launch_count(2)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        flush.fill_(1)
        step()
    torch.cuda.synchronize()
    for o in outs:
        assert int(o.status.abs().sum().item()) == 0, "a benchmark instance was rejected"

    # ---- timed region: K steps, CUDA events around each step, L2 flushed in between -----------
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches = 0
    barrier()
    t0 = time.time()
    for k in range(args.steps):
        flush.fill_(k & 0xff)
        ev[k][0].record(stream)
        launches += step()
        ev[k][1].record(stream)
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))

    # ---- per-phase times of the same step (events recorded inside the library, same stream) ---
    B.set_profiling(True)
    phase = []
    for _ in range(max(2, min(args.steps, 5))):
        flush.fill_(3)
        step(profile=phase)
    B.set_profiling(False)
    phase = np.array(phase, dtype=np.float64)            # [calls, 4]
    sim_ms = float(np.median(phase[:, 1]))               # the one k_sim_slots launch of a step (all four policies); median: one slow launch must not move it
    share = {"phase_a_keys_sort_rank": float(phase[:, 0].sum() / phase[:, 3].sum()),
             "phase_b_simulator": float(phase[:, 1].sum() / phase[:, 3].sum()),
             "phase_c_p99": float(phase[:, 2].sum() / phase[:, 3].sum())}

    # ---- end to end through the C ABI with host buffers: H2D of the trace from pinned memory,
    # the four policy runs, D2H of every output.  The batch goes through in `--e2e-chunks` chunks of
    # instances, each on its own stream (copies of one chunk overlap the simulation of the other);
    # per chunk it is the same public call as above --------------------------------------------
    n_chunks = max(1, min(args.e2e_chunks, batch.n_instances))
    bounds = [S.strong_shard(batch.n_instances, c, n_chunks) for c in range(n_chunks)]
    subs = [batch.subset(range(lo, hi)) for lo, hi in bounds]
    streams = [torch.cuda.Stream(device=dev) for _ in range(n_chunks)]
    # Per chunk ONE pinned host block and ONE device block for the five trace arrays, ONE device block
    # and ONE pinned host block for every output of every policy: a chunk is one H2D copy, one call,
    # one D2H copy (the C ABI takes plain pointers: the arrays are views into the blocks)
    IN_FIELDS = (("offsets", torch.int64), ("arrival", torch.int32), ("prompt", torch.int32), ("output", torch.int32), ("bit", torch.uint8))

    def carve(block, specs):
        """views of `block` (uint8) for (name, dtype, numel) specs, each 256-byte aligned"""
        views, off = {}, 0
        for name, dt, numel in specs:
            nbytes = numel * torch.empty(0, dtype=dt).element_size()
            views[name] = block[off: off + nbytes].view(dt)
            off += (nbytes + 255) // 256 * 256
        return views

    def block_bytes(specs):
        return sum((numel * torch.empty(0, dtype=dt).element_size() + 255) // 256 * 256 for _, dt, numel in specs)

    c_in_host, c_in_dev, c_trace, c_outs, c_out_dev, c_out_host, c_ws, host_out = [], [], [], [], [], [], [], []
    h2d = d2h = 0
    for sub in subs:
        in_specs = [(k, dt, int(getattr(sub, k).size)) for k, dt in IN_FIELDS]
        hb = torch.empty(block_bytes(in_specs), dtype=torch.uint8).pin_memory()
        db = torch.empty(block_bytes(in_specs), dtype=torch.uint8, device=dev)
        hv, dv = carve(hb, in_specs), carve(db, in_specs)
        for k, _ in IN_FIELDS:
            hv[k].copy_(torch.from_numpy(getattr(sub, k)))
        c_in_host.append(hb); c_in_dev.append(db)
        c_trace.append(B.DeviceTrace(dv["offsets"], dv["arrival"], dv["prompt"], dv["output"], dv["bit"], sub.n_instances,
                                     sub.n_requests, sub.max_n, int(sub.O0), int(sub.O1), int(sub.M)))
        h2d += int(hb.numel())
        out_specs = []
        for i in range(len(POLICIES)):
            for k in B.RESULT_FIELDS:
                dt = B._PER_REQUEST.get(k) or B._PER_INSTANCE[k]
                out_specs.append((f"{i}.{k}", dt, max(sub.n_requests if k in B._PER_REQUEST else sub.n_instances, 1)))
        ob = torch.empty(block_bytes(out_specs), dtype=torch.uint8, device=dev)
        oh = torch.empty(block_bytes(out_specs), dtype=torch.uint8).pin_memory()
        ov, ohv = carve(ob, out_specs), carve(oh, out_specs)
        c_out_dev.append(ob); c_out_host.append(oh)
        c_outs.append([B.SimOut(**{k: ov[f"{i}.{k}"] for k in B.RESULT_FIELDS}) for i in range(len(POLICIES))])
        host_out.append([{k: ohv[f"{i}.{k}"] for k in B.RESULT_FIELDS} for i in range(len(POLICIES))])
        c_ws.append(torch.empty(B.svf_simulate_policies_workspace_bytes(c_trace[-1], len(POLICIES)), dtype=torch.uint8, device=dev))
        d2h += int(oh.numel())

    def e2e_step():
        for c in range(n_chunks):
            with torch.cuda.stream(streams[c]):
                c_in_dev[c].copy_(c_in_host[c], non_blocking=True)
                B.svf_simulate_policies(c_trace[c], POLICIES, outs=c_outs[c], ws=c_ws[c])
                c_out_host[c].copy_(c_out_dev[c], non_blocking=True)
        torch.cuda.synchronize()
        return int(host_out[0][0]["total_latency"][0])

    e2e_step()
    # the chunked, eight-stream leg must give what the single call gave: every policy, every field
    for i in range(len(POLICIES)):
        for k in B.RESULT_FIELDS:
            n_k = batch.n_requests if k in ("start", "finish") else batch.n_instances
            whole = getattr(outs[i], k)[:n_k].cpu()
            parts = torch.cat([host_out[c][i][k][: (subs[c].n_requests if k in ("start", "finish") else subs[c].n_instances)]
                               for c in range(n_chunks)])
            assert torch.equal(whole, parts), f"end-to-end leg differs from the single call: policy {POLICY_NAMES[i]}, field {k}"
    barrier()
    te0 = time.perf_counter()
    n_e2e = max(2, min(args.steps, 5))
    for _ in range(n_e2e):
        e2e_step()
    barrier()
    e2e_s = (time.perf_counter() - te0) / n_e2e

    # ---- reduce over ranks: max time, summed work -------------------------------------------
    decisions = sum(int(o.decisions.sum().item()) for o in outs)
    (total_ms, e2e_s), (rs_all, dec_all, launches_all) = S.reduce_report(
        [total_ms, e2e_s], [rs_step, decisions, launches], device=dev)   # max over ranks / summed
    launches_all = int(launches_all)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- algorithmic work of the dominant kernel, counted by its counting variant (untimed) ----
    B.set_profiling(2)
    B.svf_simulate_policies(dt_dev, POLICIES, outs=outs, ws=ws)
    E, U, n_eval, n_blocked = B.simulate_work_counts()
    B.set_profiling(False)
    ops_per_launch = OPS_PER_EXAMINED * E + OPS_PER_UPDATED * U

    ms_per_step = total_ms / args.steps
    value = rs_all / (ms_per_step * 1e-3)
    hbm_peak, hbm_src = measured_peaks()
    peak_ops, peak_src = alu_peak(torch, dev)
    sim_bytes = SIM_BYTES_PER_REQUEST * batch.n_requests * len(POLICIES)
    achieved = ops_per_launch / (sim_ms * 1e-3)
    traffic, traffic_src = profiled_dram_traffic()
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int32/int64", "data": "synthetic",
        "config": workload_config(args),
        "decisions_per_sec": dec_all / (ms_per_step * 1e-3),
        "requests_per_sec": world * batch.n_requests * len(POLICIES) / (ms_per_step * 1e-3),
        "step_ms": step_ms,
        "clocks": clocks,
        "e2e": {"value": rs_all / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": 1e3 * e2e_s, "chunks": n_chunks},
        "gpu_launches": launches_all,
        "roofline": {"kernel": "k_sim_slots (persistent simulator, phase B)", "bound": "alu",
                     "achieved": achieved / 1e12, "peak": peak_ops / 1e12, "unit": "Tlane-op/s",
                     "frac": achieved / peak_ops, "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": peak_src,
                     "frac_of_integer_pipe_rate": achieved / (peak_ops / 2),   # the alu pipe alone issues every other cycle
                     "algorithmic_ops_per_launch": ops_per_launch,
                     "entries_examined_per_launch": E,
                     "entries_updated_per_launch": U,
                     "evaluations_per_launch": n_eval, "blocked_evaluations_per_launch": n_blocked,
                     "kernel_ms": sim_ms, "share_of_step": share,
                     "hbm": {"algorithmic_bytes_per_launch": sim_bytes,
                             "achieved_gbs": sim_bytes / (sim_ms * 1e-3) / 1e9, "peak_gbs": hbm_peak,
                             "frac": sim_bytes / (sim_ms * 1e-3) / 1e9 / hbm_peak, "peak_source": hbm_src},
                     "note": "integer-ALU/issue bound by design: the per-step state stays in registers, HBM only "
                             "sees the trace once (DESIGN.md 6); 'kernels' lists the HBM-bound pieces"},
    }
    peak = hbm_peak
    line["fingerprint_fnv1a64"] = T.trace_fingerprint(batch)
    # the reported CPU baseline first (oracle on the host cores), then the headline, THEN the extras:
    # nothing an extra does (an exception, a crash, a long line) can cost the line the driver reads
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args)
    extras_path = None if args.no_extras else (args.extras_file or EXTRAS_FILE)
    print(build_headline(line, extras_path), flush=True)
    if extras_path is not None:
        extras = dict(_finite(line))
        legs = (("kernels", lambda: kernel_extras(B, torch, dev, peak)),
                ("admit_sweep", lambda: admit_sweep(B, torch, dev, peak)),
                ("configs", lambda: config_extras(B, torch, dev, args, with_oracle=not (args.no_oracle_extras or args.no_cpu_baseline))),
                ("ratio_to_lower_bound", lambda: bound_extras(B, torch, dev, args)),
                ("stochastic_regime", lambda: stochastic_extras(B, torch, dev)),
                ("paper_metrics", lambda: paper_metrics_extras(B, dt_dev, outs, batch)))
        for name, leg in legs:
            try:
                extras[name] = _finite(leg())
            except Exception as e:   # recorded, never fatal: the headline is already out
                extras[name] = {"error": f"{type(e).__name__}: {e}"}
            try:
                full_path = extras_path if os.path.isabs(extras_path) else os.path.join(ROOT, extras_path)
                os.makedirs(os.path.dirname(full_path), exist_ok=True)
                with open(full_path + ".tmp", "w") as f:
                    json.dump(extras, f, indent=1)
                os.replace(full_path + ".tmp", full_path)
            except OSError as e:
                print(f"bench.py: could not write {extras_path}: {e}", file=sys.stderr)
    if world > 1:
        dist.destroy_process_group()


def paper_metrics_extras(B, dt_dev, outs, batch):
    """the paper's own metrics on the bench batch, per policy, this rank."""
    from paper_2606_22327_b200 import report as RP
    res = {name: RP.paper_metrics(dt_dev.arrival, dt_dev.output, o.finish[: batch.n_requests], dt_dev.offsets, o.status)
           for name, o in zip(POLICY_NAMES, outs)}
    res["units"] = "per-token latency in model steps per output token; throughput in tokens per step per instance"
    return res


def _finite(x):
    """Strict JSON has no Infinity / NaN: a bound that does not exist (rho >= 1) is printed as null."""
    if isinstance(x, float):
        return x if x == x and abs(x) != float("inf") else None
    if isinstance(x, dict):
        return {k: _finite(v) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_finite(v) for v in x]
    return x


def _time_cuda(torch, fn, reps=5, flush=None):
    fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        if flush is not None:
            flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); fn(); b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return float(np.mean(ts))


def kernel_extras(B, torch, dev, peak):
    """The HBM-bound subsystems timed alone (inputs larger than L2: 2^26 requests)."""
    out = []
    n = 1 << 26
    g = torch.Generator(device=dev); g.manual_seed(1)
    s = torch.randint(16, 8193, (n,), device=dev, dtype=torch.int32, generator=g)
    o = torch.randint(1, 4097, (n,), device=dev, dtype=torch.int32, generator=g)
    words = torch.empty(n, dtype=torch.int64, device=dev)
    st = torch.empty(1, dtype=torch.int32, device=dev)
    ms = _time_cuda(torch, lambda: B.svf_keys(B.SVF, s, o, None, None, 1, 1, words, st))
    bytes_keys = n * (4 + 4 + 8)
    out.append({"kernel": "svf_keys (policy svf, n=2^26)", "ms": ms, "achieved": bytes_keys / ms / 1e6, "unit": "GB/s",
                "frac": bytes_keys / ms / 1e6 / peak, "algorithmic_bytes": bytes_keys})
    srt = torch.empty_like(words)
    wsb = torch.empty(int(B.lib().svf_sort_workspace_bytes(n, 32, 64)), dtype=torch.uint8, device=dev)
    ms = _time_cuda(torch, lambda: B.svf_sort_words(words, 32, 64, out=srt, ws=wsb), reps=3)
    # keys < 2^26: 4 executed passes of the 4 planned (max key 8192*4096+4096*4097/2 needs 26 bits)
    bytes_sort = n * (8 + 16 * 4)
    out.append({"kernel": "svf_sort_words (n=2^26, key bits [32,64), 4 passes executed)", "ms": ms,
                "achieved": bytes_sort / ms / 1e6, "unit": "GB/s", "frac": bytes_sort / ms / 1e6 / peak,
                "algorithmic_bytes": bytes_sort, "words_per_sec": n / ms * 1e3})
    return out


def admit_sweep(B, torch, dev, peak):
    """the stateless admission decision at depth.  W waiting requests (BASELINE.json
    configs[3] laws) x R running requests (a loaded engine: the running set alone peaks at 0.8 M),
    M = 1e6, policy SVF; the phase split comes from CUDA events the library records on the stream."""
    res = []
    M = 1_000_000
    for W, runs in ((1 << 10, (256, 1024, 4096)), (1 << 14, (256, 1024, 4096)), (1 << 18, (256, 1024, 4096)),
                    (1 << 20, (1024,)), (1 << 22, (1024,))):         # the last two: queues beyond L2, where bandwidth starts to count
        for R in runs:
            w_s, w_o, w_a, w_bit, r_kv, r_rem = T.admit_state(W + R, W, R, M)
            d = [torch.from_numpy(np.ascontiguousarray(x)).to(dev) for x in (w_s, w_o, w_a, w_bit, r_kv, r_rem)]
            ws = torch.empty(B.svf_admit_workspace_bytes(W, R), dtype=torch.uint8, device=dev)
            out = B.svf_admit(B.SVF, M, 0, d[0], d[1], d[2], d[3], 179, 887, d[4], d[5], ws=ws)
            call = lambda: B.svf_admit(B.SVF, M, 0, d[0], d[1], d[2], d[3], 179, 887, d[4], d[5], ws=ws, out=out)
            ms = _time_cuda(torch, call, reps=10)
            B.set_profiling(True)
            ph = []
            for _ in range(5):
                call()
                ph.append(B.admit_phase_ms())
            B.set_profiling(False)
            ph = np.array(ph).mean(axis=0)
            k = int(out.n_admitted.item())
            # a deep call is a chain of 13 small launches: the same call captured once in a CUDA graph and
            # replayed (what a caller that decides every engine step would do); same buffers, same answer
            graph_ms = None
            if W + R > 8192:
                try:
                    side = torch.cuda.Stream(device=dev)
                    with torch.cuda.stream(side):
                        call()
                    torch.cuda.synchronize()
                    graph = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(graph, stream=side):
                        call()
                    out.n_admitted.fill_(-1)
                    graph_ms = _time_cuda(torch, graph.replay, reps=10)
                    if int(out.n_admitted.item()) != k:
                        graph_ms = f"replay gave {int(out.n_admitted.item())} admitted, the direct call {k}"
                    del graph
                except Exception as e:      # an extra: recorded, never fatal
                    graph_ms = f"{type(e).__name__}: {e}"
            # what the call must move: validation + keys read s, o, a (12 B) and write the packed word
            # (8 B); the sort reads the words once for its histograms and reads + writes them once per
            # executed pass (26-bit keys: four 8-bit passes over [32, 64)); the sorted words are copied
            # out (16 B); the admission reads the running set and the first candidates (12 B each)
            fused = W + R <= 8192          # the library then takes the whole decision in ONE launch on one CTA
            algo = (W * (12 + 8 + 4) + R * 8) if fused else W * (12 + 8 + 8 + 16 * 4 + 16) + (R + min(W, 8192 - R)) * 12
            res.append({"W": W, "R": R, "ms": ms, "ms_replayed_from_a_cuda_graph": graph_ms, "admitted": k, "launches": B.last_launch_count(1),
                        "decisions_per_sec": (k + 1) / ms * 1e3, "queue_entries_per_sec": W / ms * 1e3,
                        "phase_ms": {"keys_and_validation": float(ph[0]), "sorts": float(ph[1]), "admission": float(ph[2]),
                                     "whole_call_under_events": float(ph[3])},
                        # at these sizes the call is a short chain of small launches (or one CTA): latency, not
                        # bandwidth, sets the time; the bytes are reported as a rate, without an HBM fraction
                        "roofline": {"bound": "hbm", "achieved": algo / ms / 1e6, "peak": peak, "unit": "GB/s", "frac": algo / ms / 1e6 / peak,
                                     "algorithmic_bytes": algo, "note": "queue beyond L2: keys + four onesweep passes over the whole queue set the time"}
                                    if W >= 1 << 20 else
                                    {"bound": "latency", "achieved": algo / ms / 1e6, "unit": "GB/s", "algorithmic_bytes": algo,
                                     "note": ("one launch, one CTA: validation, keys, both sorts and the bisection in shared memory (the phase "
                                              "split does not apply: all under 'admission'); bound by one SM's issue rate and barriers") if fused else
                                             "a chain of 13 small launches: launch latency, not bandwidth, sets the time at these sizes"}})
    return res


def _oracle_ms(svf_ref, tr, policy, threads):
    t0 = time.perf_counter()
    r = svf_ref.simulate(tr, policy, n_threads=threads)
    return 1e3 * (time.perf_counter() - t0), r


def config_extras(B, torch, dev, args, with_oracle=True):
    """Every BASELINE.json config at its stated size, device resident, with the oracle timed beside it
    on the host cores of the same box: one core for the single-instance configs, all
    cores plus the one-core figure (on a sample) for the batched ones.  Context, not the headline."""
    svf_ref, threads = None, 1
    if with_oracle:
        from oracle import svf_ref
        svf_ref.build()
        threads = min(os.cpu_count() or 1, svf_ref.max_threads())
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    info = {"nproc": os.cpu_count(), "oracle_threads_all_cores": threads, "entries": []}

    def gpu_run(tr, pols):
        d = B.DeviceTrace.from_host(tr, device=dev)
        outs = [B.SimOut.alloc(d) for _ in pols]
        ws = torch.empty(B.svf_simulate_policies_workspace_bytes(d, len(pols)), dtype=torch.uint8, device=dev)
        ms = _time_cuda(torch, lambda: B.svf_simulate_policies(d, pols, outs=outs, ws=ws), reps=3, flush=flush)
        return ms, outs

    def entry(name, tr, pols, ms, outs, oracle=None):
        e = {"config": name, "policies": [POLICY_NAMES[p] for p in pols], "gpu_ms": ms,
             "instances": tr.n_instances, "requests": tr.n_requests, "M": tr.M, "fingerprint_fnv1a64": T.trace_fingerprint(tr),
             "request_steps_per_sec": tr.request_steps * len(pols) / ms * 1e3,
             "decisions_per_sec": sum(int(o.decisions.sum().item()) for o in outs) / ms * 1e3,
             "total_latency": {POLICY_NAMES[p]: int(o.total_latency.sum().item()) for p, o in zip(pols, outs)}}
        if oracle:
            e["oracle"] = oracle
        info["entries"].append(e)
        return e

    def check(name, pol, out, ref):
        assert int(out.total_latency.sum().item()) == int(ref.total_latency.sum()), f"{name}: GPU and oracle disagree ({POLICY_NAMES[pol]})"

    # configs[0]: n = 8 at t = 0, M = 32; 512 seeded instances in one batch
    tr = T.concat([T.config1(i) for i in range(512)], "cfg1x512", 32, 2, 8)
    ms, outs = gpu_run(tr, list(POLICIES))
    orc = None
    if svf_ref:
        oms = [_oracle_ms(svf_ref, tr, p, 1) for p in POLICIES]
        for p, (_, r) in zip(POLICIES, oms):
            check("configs[0]", p, outs[p], r)
        orc = {"ms_1_core": sum(m for m, _ in oms), "cores": 1, "sample": "the same 512 instances x 4 policies"}
    entry("configs[0] tiny offline instance, 512 seeds", tr, list(POLICIES), ms, outs, orc)

    # configs[1]: one online trace, n = 2,000
    tr = T.config2(0)
    for p in POLICIES:
        ms, outs = gpu_run(tr, [p])
        orc = None
        if svf_ref:
            oms, r = _oracle_ms(svf_ref, tr, p, 1)
            check("configs[1]", p, outs[0], r)
            orc = {"ms_1_core": oms, "cores": 1, "sample": "the same trace"}
        e = entry("configs[1] single online trace n=2000", tr, [p], ms, outs, orc)
        e["p99_latency"] = int(outs[0].p99_latency[0].item())

    # configs[2]: 4,096 x 1,000 at rates 2, 4, 8: four policies per call
    for lam in (2.0, 4.0, 8.0):
        tr = T.config3(n_instances=args.instances, n=args.requests, lam=lam)
        ms, outs = gpu_run(tr, list(POLICIES))
        orc = None
        if svf_ref:
            t0 = time.perf_counter()
            refs = [svf_ref.simulate(tr, p, n_threads=threads) for p in POLICIES]
            all_ms = 1e3 * (time.perf_counter() - t0)
            for p, r in zip(POLICIES, refs):
                check(f"configs[2] rate {lam:g}", p, outs[p], r)
            sub = tr.subset(range(0, tr.n_instances, max(1, tr.n_instances // 64)))
            one_ms = sum(_oracle_ms(svf_ref, sub, p, 1)[0] for p in POLICIES)
            orc = {"ms_all_cores": all_ms, "cores": threads, "sample": "the same batch x 4 policies",
                   "ms_1_core_scaled": one_ms * tr.n_instances / sub.n_instances,
                   "one_core_sample": f"{sub.n_instances} of {tr.n_instances} instances x 4 policies, scaled by the instance count"}
        entry(f"configs[2] batched simulation, Poisson rate {lam:g}", tr, list(POLICIES), ms, outs, orc)

    # configs[3]: one instance of 200,000 requests: a single serial step chain
    tr = T.config4()
    refs4 = None
    if svf_ref:
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(len(POLICIES)) as ex:          # each policy alone on one core, side by side
            refs4 = list(ex.map(lambda p: _oracle_ms(svf_ref, tr, p, 1), POLICIES))
    for p in POLICIES:
        ms, outs = gpu_run(tr, [p])
        orc = None
        if refs4:
            check("configs[3]", p, outs[0], refs4[p][1])
            orc = {"ms_1_core": refs4[p][0], "cores": 1, "sample": "the same trace (the four policies timed side by side, one core each)"}
        entry("configs[3] high-concurrency single instance n=200000", tr, [p], ms, outs, orc)

    # configs[4]: 256 x 5,000, bimodal outputs: the (M, p) grid under SVF, 1-bit SVF, SJF
    pols5 = [B.SVF, B.SVF_1BIT, B.SJF]
    for M in (50_000, 200_000, 800_000):
        for pf in (0.0, 0.05, 0.2):
            tr = T.config5(M=M, p_flip=pf)
            ms, outs = gpu_run(tr, pols5)
            orc = None
            if svf_ref:
                t0 = time.perf_counter()
                refs = [svf_ref.simulate(tr, p, n_threads=threads) for p in pols5]
                all_ms = 1e3 * (time.perf_counter() - t0)
                for p, o_, r in zip(pols5, outs, refs):
                    check(f"configs[4] M={M} p={pf:g}", p, o_, r)
                orc = {"ms_all_cores": all_ms, "cores": threads, "sample": "the same batch x 3 policies"}
                if pf == 0.0:
                    sub = tr.subset(range(0, tr.n_instances, 32))
                    one_ms = sum(_oracle_ms(svf_ref, sub, p, 1)[0] for p in pols5)
                    orc["ms_1_core_scaled"] = one_ms * tr.n_instances / sub.n_instances
                    orc["one_core_sample"] = f"{sub.n_instances} of {tr.n_instances} instances x 3 policies, scaled by the instance count"
            entry(f"configs[4] 1-bit SVF sweep M={M} p={pf:g}", tr, pols5, ms, outs, orc)
    return info


def stochastic_extras(B, torch, dev):
    """the stochastic regime of PAPER.md 3.4 / App. H on the GPU: Poisson arrivals,
    o ~ Geo(1/293) (truncated at 4,096), prompts as configs[1], M = 300,000.  E[TEL] per request is
    estimated over 256 instances x 2,000 requests per policy, divided by Lemma H.1's lower bound on
    E[TEL(OPT)] (Eq. 89) and set beside the bounds of Thm 3.4 (Eq. 7) and Thm 3.5 (Eq. 8); the sweep over
    the 1-bit threshold theta shows the gap closing as eps decays (Remark).  Float report
    layer (report.py), outside the parity contract; finite runs start empty, so they sit below the
    steady state the theorems are about."""
    from paper_2606_22327_b200 import report as RP
    mu, M, p_max, I, n = 1.0 / 293.0, 300_000, 4096 + 4096, 256, 2000
    res = {"workload": f"{I} instances x {n} requests, o ~ Geo(1/293) truncated at 4096, M = {M}, alpha = p_max/M = {p_max / M:.4f}",
           "load_sweep": [], "theta_sweep": []}

    def run(tr, pols):
        d = B.DeviceTrace.from_host(tr, device=dev)
        outs = B.svf_simulate_policies(d, pols, want=("total_latency", "status"))
        torch.cuda.synchronize()
        return [RP.mean_request_latency(o.total_latency, d.offsets, o.status) for o in outs]

    mean_s = float(T.stochastic(n_instances=I, n=n, lam=1.0, M=M).prompt.mean())
    # rho is the paper's CONSERVATIVE load: rho = 1 is about half of the raw volume capacity M per step,
    # so inside the theorems' range (rho < 1) hardly anybody waits and every policy sits at the lower
    # bound; 2.5 and 4 are outside it (transient overload while the arrivals last; no bound: null)
    # and show where the policies part
    for rho in (0.3, 0.6, 0.9, 2.5, 4.0):
        lam = RP.rate_for_load(rho, mu, mean_s, M, p_max)
        tr = T.stochastic(n_instances=I, n=n, lam=lam, M=M)
        c = RP.stochastic_constants(mu, mean_s, lam, M, p_max, theta=293)
        lat = run(tr, list(POLICIES))
        res["load_sweep"].append({"rho": rho, "lambda": lam, "opt_lower_bound": c["opt_lower_bound"],
                                  "thm34_bound": c["thm34_bound"], "thm35_bound_theta293": c["thm35_bound"],
                                  "mean_latency": dict(zip(POLICY_NAMES, lat)),
                                  "ratio_to_opt_lower_bound": {k: v / c["opt_lower_bound"] for k, v in zip(POLICY_NAMES, lat)},
                                  "svf_below_thm34": lat[0] / c["opt_lower_bound"] <= c["thm34_bound"],
                                  "onebit_below_thm35": lat[1] / c["opt_lower_bound"] <= c["thm35_bound"]})
    for rho, theta in [(r_, th) for r_ in (0.9, 4.0) for th in (64, 147, 293, 586)]:
        lam = RP.rate_for_load(rho, mu, mean_s, M, p_max)
        tr = T.stochastic(n_instances=I, n=n, lam=lam, M=M, theta=theta)
        c = RP.stochastic_constants(mu, mean_s, lam, M, p_max, theta=theta)
        lat = run(tr, [B.SVF_1BIT, B.SVF])
        res["theta_sweep"].append({"rho": rho, "theta": theta, "O0": tr.O0, "O1": tr.O1, "eps": c["eps"], "E_vol": c["E_vol"],
                                   "thm35_bound": c["thm35_bound"], "thm34_bound": c["thm34_bound"],
                                   "ratio_1bit": lat[0] / c["opt_lower_bound"], "ratio_svf": lat[1] / c["opt_lower_bound"],
                                   "onebit_below_thm35": lat[0] / c["opt_lower_bound"] <= c["thm35_bound"]})
    return res


def bound_extras(B, torch, dev, args):
    """the burst version of the bench batch (all arrivals at 0): TEL(policy) * M
    over the volume lower bound of Prop. 3.1 -- an upper bound on each policy's approximation
    ratio where the optimum cannot be computed (Thm 3.2 bounds SVF's true ratio by 1 + 2/(1-alpha))."""
    tr = T.config3(n_instances=min(args.instances, 4096), n=args.requests, lam=args.lam)
    tr.arrival[:] = 0
    d = B.DeviceTrace.from_host(tr, device=dev)
    ms = _time_cuda(torch, lambda: B.svf_volume_lower_bound(d), reps=3)
    lb, st = B.svf_volume_lower_bound(d)
    outs = B.svf_simulate_policies(d, POLICIES, want=("total_latency", "status"))
    torch.cuda.synchronize()
    lbf = lb.double()
    res = {"workload": f"burst version of the bench batch ({tr.n_instances} x {args.requests}, all arrivals at t=0)",
           "lower_bound_ms": ms, "lower_bound_status_ok": bool(int(st.abs().sum().item()) == 0)}
    for name, out in zip(POLICY_NAMES, outs):
        r = out.total_latency.double() * float(tr.M) / lbf
        res[name] = {"mean": float(r.mean().item()), "max": float(r.max().item())}
    return res


def cpu_baseline(args):
    from oracle import svf_ref
    svf_ref.build()
    threads = min(os.cpu_count() or 1, svf_ref.max_threads())
    n_inst = args.instances
    sample = T.config3(n_instances=n_inst, n=args.requests, lam=args.lam)
    oracle_step(svf_ref, sample.subset(range(min(8, n_inst))), threads)
    t0 = time.perf_counter()
    reps = 0
    while True:
        oracle_step(svf_ref, sample, threads)
        reps += 1
        if time.perf_counter() - t0 > 12.0 or reps >= 40:
            break
    dt = time.perf_counter() - t0
    return {"value": sample.request_steps * len(POLICIES) * reps / dt, "unit": UNIT, "cores": threads,
            "kind": "oracle", "nproc": os.cpu_count(),
            "sample": f"all {n_inst} instances x {args.requests} requests x 4 policies (rank 0's batch), "
                      f"{reps} repetitions, {dt:.1f} s, instance-parallel over {threads} host threads"}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
