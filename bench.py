"""bench.py -- one JSON line per run for the H-ADPSGD super-learner step.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload swb2000] [--impl reference]

A "step" is one pass of the whole hot path (pairing, learner mean,
momentum SGD, pairwise mix, diagnostics) = ONE fused kernel launch over one batch of synthetic
gradients.  Metric (BASELINE.json): learner-params updated per second = S*G*P / t_step, with
the achieved HBM GB/s in `roofline`.  Default workload = BASELINE.json configs[2], the
145,145,344-parameter SWB-2000-shaped flat fp32 buffer with S=16 super-learners x G=4
learners (55.7 GB resident), which is the configuration the metric is quoted on.

N > 1 (torchrun): the path is element-wise independent, so every rank owns one P-element
range of an N*P-parameter model (no data-path collective, "scaling": "weak"); only the few
diagnostic doubles are all-reduced, after the timed region.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload on the host cores; rank 0 only.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "learner_params_updated_per_sec"
UNIT = "learner-params/s"
LR, MU = 0.1, 0.9
FALLBACK_HBM_GBS = 6650.0       # /opt/skills/guides/B200_PROFILING.md fallback
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the step kernel, from the
# `ncu --set full` capture summarised in profiles/ (bytes; None until a capture exists)
NCU_TRAFFIC_BYTES = {"swb2000": 74.284e9, "swb300": 48.502e9, "swb2000_ragged_bf16": 37.123e9, "paper_literal": 16.536e9}
NCU_TRAFFIC_SHARED = {"swb2000": 66.555e9, "swb2000_ragged_bf16": 33.285e9}     # same, with HADPSGD_SHARE_PAIR_WEIGHTS (profiles/r01_share_pair_weights.md)
NCU_TRAFFIC_SOURCE = {"swb2000": "profiles/r01_step_kernel_ncu.md (dram__bytes_read.sum 55.737 GB + dram__bytes_write.sum 18.545 GB)",
                      "swb300": "profiles/r01_traffic_other_workloads.md", "swb2000_ragged_bf16": "profiles/r01_traffic_other_workloads.md",
                      "paper_literal": "profiles/r01_traffic_other_workloads.md"}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="swb2000")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample-elems", type=int, default=1 << 22)
    ap.add_argument("--cpu-sample-steps", type=int, default=20)
    ap.add_argument("--blocks-per-sm", type=int, default=0)
    ap.add_argument("--flags", default="", help="comma list: deterministic,no_diag,no_mix,eq7,share")
    ap.add_argument("--no-share-leg", action="store_true", help="skip the extra HADPSGD_SHARE_PAIR_WEIGHTS leg")
    ap.add_argument("--emit-bf16", action="store_true",
                    help="also write the bf16 working copy of the weights every step (row f2; +2 B/param)")
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE.json configs[4]: bandwidth sweep over P, S, G (one JSON line per point)")
    ap.add_argument("--sweep-md", default="", help="also write the sweep as a markdown table to this path")
    return ap.parse_args()


def workload(name):
    from fixtures import shapes
    cfg = dict(shapes.CONFIGS[name])
    cfg["P"] = int(sum(cfg["seg_len"]))
    cfg["b_g"] = 2 if cfg["grad"] == "bf16" else 4
    return cfg


def algorithmic_bytes(cfg):
    """per parameter per super-learner, read G*b_g + 4 (w) + 4 (v), write 4 + 4
    (+ 2 when the bf16 working copy is emitted)."""
    return cfg["S"] * cfg["P"] * (cfg["G"] * cfg["b_g"] + 16 + (2 if cfg.get("emit") else 0))


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, STREAM-style copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------ clocks during the timed region

class ClockSampler:
    """SM clock and throttle reasons DURING the timed region: an NVML polling thread (every few
    ms; the timed loop spends its time inside cudaDeviceSynchronize, which releases the GIL).
    Falls back to one `nvidia-smi` query loop (the recipe's clocks line) if NVML is unusable."""
    QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None
        self.thread, self.stop_flag, self.samples, self.bits, self.max_mhz, self.power = None, False, [], 0, None, []

    def _poll(self, nv, dev):
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(dev, nv.NVML_CLOCK_SM))
                self.bits |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(dev))
                self.power.append(nv.nvmlDeviceGetPowerUsage(dev) / 1000.0)
            except Exception:
                pass
            time.sleep(0.004)

    def start(self):
        try:
            import threading
            import pynvml as nv
            nv.nvmlInit()
            dev = nv.nvmlDeviceGetHandleByIndex(self._physical_index())
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(dev, nv.NVML_CLOCK_SM)
            self.thread = threading.Thread(target=self._poll, args=(nv, dev), daemon=True)
            self.thread.start()
            return
        except Exception:
            self.thread = None
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self._physical_index()), "--query-gpu=" + self.QUERY,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=fd, stderr=subprocess.DEVNULL)
            os.close(fd)
        except Exception:
            self.proc = None

    def _physical_index(self):
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            ids = [x for x in vis.split(",") if x.strip()]
            if self.index < len(ids) and ids[self.index].strip().isdigit():
                return int(ids[self.index])
        return self.index

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "source": None}
        if self.thread is not None:
            self.stop_flag = True
            self.thread.join(timeout=2)
            sm = sorted(self.samples)
            if sm:
                out.update(sm_mhz=float(sm[len(sm) // 2]), sm_max_mhz=float(self.max_mhz), samples=len(sm), source="nvml",
                           power_w_max=max(self.power) if self.power else None)
            out["reasons"] = sorted(name for bit, name in self.REASONS.items() if self.bits & bit)
            return out
        if self.proc is None:
            return out
        self.proc.terminate()           # the exact PID we started
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1])); mx.append(float(f[2]))
                except ValueError:
                    continue
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), samples=len(sm), source="nvidia-smi")
        out["reasons"] = sorted(reasons)
        return out


# ------------------------------------------------------------------ CPU oracle legs

def host_cpu():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except Exception:
        pass
    return model, os.cpu_count()


def time_oracle(cfg, n_elems, steps, warmup=1):
    """The oracle as it stands (single thread, oracle/hadpsgd_oracle.cpp) on a bounded sample:
    the first n_elems parameters of every buffer of the workload (the method is element-wise
    independent, so a window is the same work per parameter).  Returns seconds per step."""
    import numpy as np
    import oracle
    from fixtures import problem
    S, G = cfg["S"], cfg["G"]
    n = min(n_elems, cfg["P"])
    bf16 = cfg["grad"] == "bf16"
    w = problem.host_weights(7, S, 0, n)
    v = np.zeros((S, n), np.float32)
    g = problem.host_grads(7, 0, S, G, 0, n, cfg["dist"], bf16=bf16)
    for k in range(warmup):
        oracle.step(g, w, v, LR, MU, k, diag=True)
    t0 = time.perf_counter()
    for k in range(steps):
        oracle.step(g, w, v, LR, MU, warmup + k, diag=True)
    dt = (time.perf_counter() - t0) / max(steps, 1)
    return dt, n


def cpu_baseline(cfg, n_elems, steps):
    dt, n = time_oracle(cfg, n_elems, steps)
    model, ncpu = host_cpu()
    return {"value": cfg["S"] * cfg["G"] * n / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"first {n} of {cfg['P']} params of every buffer (S={cfg['S']}, G={cfg['G']}), "
                      f"{steps} steps after 1 warm-up, diagnostics on; single thread; host has {ncpu} logical CPUs ({model})",
            "gb_per_s": cfg["S"] * n * (cfg["G"] * cfg["b_g"] + 16) / dt / 1e9,
            "ms_per_step_sample": dt * 1e3}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = workload(args.workload)
    dt, n = time_oracle(cfg, args.cpu_sample_elems, args.steps, warmup=min(args.warmup, 2))
    model, ncpu = host_cpu()
    value = cfg["S"] * cfg["G"] * n / dt
    sample = (f"each step = first {n} of {cfg['P']} params of every buffer (S={cfg['S']}, G={cfg['G']}); "
              f"single thread; host has {ncpu} logical CPUs ({model})")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "S": cfg["S"], "G": cfg["G"], "P": cfg["P"],
                       "grad_dtype": cfg["grad"], "sample_params": n},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------ the GPU arm

def parse_flags(H, text):
    table = {"deterministic": H.DETERMINISTIC, "no_diag": H.NO_DIAG, "no_mix": H.NO_MIX, "eq7": H.EQ7_LITERAL,
             "share": H.SHARE_PAIR_WEIGHTS}
    flags = 0
    for name in filter(None, (t.strip() for t in text.split(","))):
        flags |= table[name]
    return flags


def time_device_steps(torch, dist, h, steps, warmup, k0=0, sampler=None):
    """W untimed steps, then exactly K steps between barrier + synchronize; CUDA events on the
    stream the kernel is launched on (the handle's stream IS torch's current stream)."""
    for k in range(warmup):
        h.hadpsgd_step(LR, MU, k0 + k)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if sampler is not None:
        sampler.start()
    ev0.record(h.stream)
    for k in range(steps):
        h.hadpsgd_step(LR, MU, k0 + warmup + k)
    ev1.record(h.stream)
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler is not None else None
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    return ev0.elapsed_time(ev1) / 1e3, clocks      # seconds for K steps


def time_e2e_steps(torch, dist, h, cfg, steps, warmup=1):
    """End to end through hadpsgd_step_host: every step copies all S*G gradient buffers from
    pinned HOST memory to HBM (chunked, overlapped with the kernel) and reads the diagnostics
    back to the host.  Returns (seconds for `steps` steps, h2d bytes/step, d2h bytes/step, note)."""
    S, G = cfg["S"], cfg["G"]
    nbytes = h.P_padded * cfg["b_g"]
    avail = 0
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable"):
                avail = int(line.split()[1]) * 1024
    except Exception:
        pass
    world = dist.get_world_size() if dist is not None else 1
    n_host = S * G
    # distinct pinned buffers for every learner when host RAM allows; otherwise one buffer per
    # learner index g shared by all super-learners (same bytes cross PCIe either way)
    if world > 1 or (avail and n_host * nbytes > 0.5 * avail):
        n_host = G        # N ranks share one host: keep the pinned footprint at G buffers per rank
    host = []
    for b in range(n_host):
        t = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
        src = h.hadpsgd_grads(b // G if n_host == S * G else 0, b % G)
        t.copy_(src.view(torch.uint8), non_blocking=True)
        host.append(t)
    torch.cuda.synchronize()
    ptrs = [host[(s * G + g) if n_host == S * G else g].data_ptr() for s in range(S) for g in range(G)]
    for k in range(warmup):
        h.hadpsgd_step_host(ptrs, LR, MU, k)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(h.stream)
    t0 = time.perf_counter()
    for k in range(steps):
        d = h.hadpsgd_step_host(ptrs, LR, MU, warmup + k)      # syncs: diagnostics land on the host
    ev1.record(h.stream)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    if dist is not None:
        dist.barrier()
    dev = ev0.elapsed_time(ev1) / 1e3
    assert d["gsq"].shape[0] == S
    note = f"{n_host} distinct pinned host buffers of {nbytes} B"
    return max(dev, wall), S * G * nbytes, 3 * S * 8, note


def run_ours(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback (use --impl reference for the oracle)")
    import paper_1907_05701_b200 as H
    from fixtures import problem
    H.lib()                                   # fail loudly if libhadpsgd.so is missing

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1 or "RANK" in os.environ:          # launched by torch.distributed.run (any N)
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    assert world == args.gpus, f"--gpus {args.gpus} but WORLD_SIZE={world} (launch N>1 with torch.distributed.run)"

    cfg = workload(args.workload)
    cfg["emit"] = args.emit_bf16
    S, G, P = cfg["S"], cfg["G"], cfg["P"]
    flags = parse_flags(H, args.flags)
    h = H.Hadpsgd(S, G, cfg["seg_len"], H.BF16 if cfg["grad"] == "bf16" else H.F32, flags, device=local,
                  working_dtype=H.BF16 if args.emit_bf16 else H.F32)
    if args.blocks_per_sm:
        h.hadpsgd_set_launch(args.blocks_per_sm)
    # rank r owns parameters [r*P, (r+1)*P) of an N*P-parameter model: its own seed stream
    seed = 2000 + rank
    problem.fill_weights(h, seed)
    problem.fill_grads(h, seed, 0, cfg["dist"])
    torch.cuda.synchronize()

    n0 = h.hadpsgd_launch_count()
    secs, clocks = time_device_steps(torch, dist, h, args.steps, args.warmup,
                                     sampler=ClockSampler(local) if rank == 0 else None)
    launches = h.hadpsgd_launch_count() - n0 - args.warmup
    # a timed region that saw a hardware or thermal slowdown is rejected and measured again, once
    bad = {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
    redo = torch.tensor([1 if (clocks and bad & set(clocks["reasons"])) else 0], device="cuda")
    if dist is not None:
        dist.broadcast(redo, src=0)
    remeasured = bool(int(redo[0]))
    if remeasured:
        time.sleep(5.0)
        n0 = h.hadpsgd_launch_count()
        secs, clocks = time_device_steps(torch, dist, h, args.steps, args.warmup, k0=args.steps + args.warmup,
                                         sampler=ClockSampler(local) if rank == 0 else None)
        launches = h.hadpsgd_launch_count() - n0 - args.warmup
    if clocks is not None:
        clocks["remeasured_after_slowdown"] = remeasured
    diag = None if (flags & H.NO_DIAG) else h.hadpsgd_diagnostics()

    e2e = None
    if not args.no_e2e:
        e_secs, h2d, d2h, note = time_e2e_steps(torch, dist, h, cfg, args.e2e_steps)
        e2e = (e_secs, h2d, d2h, note)

    # max over ranks (device time), diagnostics summed over the parameter shards
    if dist is not None:
        from paper_1907_05701_b200 import sharding
        secs = sharding.max_over_ranks(secs, dist, "cuda")
        if e2e:
            e2e = (sharding.max_over_ranks(e2e[0], dist, "cuda"),) + e2e[1:]
        if diag is not None:
            # the only collective: 3*S doubles, outside the timed region
            diag = sharding.allreduce_diagnostics(diag, dist, "cuda")
    arena_bytes = h.arena_bytes
    h.close()
    del h
    torch.cuda.empty_cache()

    # Second device-timed leg, reported beside the headline (never instead of it): the same step with
    # HADPSGD_SHARE_PAIR_WEIGHTS, where pair members share one weight buffer (same arithmetic and
    # results; one weight write per pair and one HBM fetch of the buffer two pairs read).
    shared = None
    can_share = not (flags & (H.NO_MIX | H.EQ7_LITERAL | H.SHARE_PAIR_WEIGHTS)) and S > 1 and S % 2 == 0
    if can_share and not args.no_share_leg:
        hs = H.Hadpsgd(S, G, cfg["seg_len"], H.BF16 if cfg["grad"] == "bf16" else H.F32, flags | H.SHARE_PAIR_WEIGHTS,
                       device=local, working_dtype=H.BF16 if args.emit_bf16 else H.F32)
        problem.fill_weights(hs, seed)
        problem.fill_grads(hs, seed, 0, cfg["dist"])
        torch.cuda.synchronize()
        s_secs, _ = time_device_steps(torch, dist, hs, args.steps, args.warmup)
        if dist is not None:
            from paper_1907_05701_b200 import sharding
            s_secs = sharding.max_over_ranks(s_secs, dist, "cuda")
        shared = s_secs / args.steps
        hs.close()
        del hs
        torch.cuda.empty_cache()

    if rank == 0:
        t_step = secs / args.steps
        peak, peak_src = measured_peak()
        abytes = algorithmic_bytes(cfg)
        achieved = abytes / t_step / 1e9
        line = {
            "metric": METRIC, "value": world * S * G * P / t_step, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_step * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "S": S, "G": G, "P": P, "n_segments": len(cfg["seg_len"]),
                       "grad_dtype": cfg["grad"], "master_dtype": "f32",
                       "working_dtype": "bf16" if args.emit_bf16 else "f32", "lr": LR, "momentum": MU,
                       "resident_bytes_per_gpu": arena_bytes, "flags": args.flags or "default (diagnostics on)",
                       "l2": "inputs larger than L2 (working set per step >> 126 MB); no flush needed",
                       "parallelism": "single GPU" if world == 1 else f"parameter-range shards x{world}, no data-path collective"},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None if args.emit_bf16 else NCU_TRAFFIC_BYTES.get(args.workload),
                         "traffic_source": None if args.emit_bf16 else NCU_TRAFFIC_SOURCE.get(args.workload),
                         "peak_source": peak_src, "algorithmic_bytes_per_launch": abytes,
                         "kernel": "hadpsgd::step_kernel (one launch = one step)", "frac_of_8TBps_nominal": achieved / 8000.0},
            "clocks": clocks, "gpu_launches": launches,
        }
        if shared is not None:
            line["share_pair_weights"] = {
                "flag": "HADPSGD_SHARE_PAIR_WEIGHTS (opt-in; bench.py --flags share makes it the headline leg)",
                "ms_per_step": shared * 1e3, "value": world * S * G * P / shared, "unit": UNIT,
                "achieved_algorithmic_gbs": abytes / shared / 1e9, "frac_of_peak_algorithmic": abytes / shared / 1e9 / peak,
                "bytes_moved_model": S * P * (cfg["G"] * cfg["b_g"] + 12 + (1 if args.emit_bf16 else 0)),
                "traffic": NCU_TRAFFIC_SHARED.get(args.workload) if not args.emit_bf16 else None,
                "note": "same arithmetic and results (parity-tested at full size); pair members share one of the S weight "
                        "buffers: 4 B less written and 4 B less fetched from HBM per pair-parameter than the algorithmic "
                        "S*P*(G*b_g+16), so achieved_algorithmic_gbs exceeds the DRAM rate actually sustained"}
        if e2e:
            e_step = e2e[0] / args.e2e_steps
            line["e2e"] = {"value": world * S * G * P / e_step, "unit": UNIT, "h2d_bytes_per_step": e2e[1],
                           "d2h_bytes_per_step": e2e[2], "ms_per_step": e_step * 1e3, "steps": args.e2e_steps,
                           "note": "hadpsgd_step_host: " + e2e[3]}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(cfg, args.cpu_sample_elems, args.cpu_sample_steps)
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_sweep(args):
    """BASELINE.json configs[4]: flat fp32 buffer of 2^10..2^28 params (powers of 4), G in {2,4,8},
    S in {2,4,8,16} with S*G*P*4 B <= 96 GB; uniform grads in [-1e-3, 1e-3]; W warm + K timed steps
    per point (defaults 5 + 20); GB/s (algorithmic) vs buffer size.  Small points are L2-resident
    (working set < 126 MB) and launch-latency bound: they are flagged, not bandwidth claims."""
    import torch
    import paper_1907_05701_b200 as H
    from fixtures import problem, shapes
    H.lib()
    torch.cuda.set_device(0)
    peak, peak_src = measured_peak()
    rows = []
    for P, S, G in shapes.sweep_points():
        h = H.Hadpsgd(S, G, [P], H.F32, parse_flags(H, args.flags), device=0)
        problem.fill_weights(h, 3000)
        problem.fill_grads(h, 3000, 0, "uniform")
        torch.cuda.synchronize()
        secs, _ = time_device_steps(torch, None, h, args.steps, args.warmup)
        t = secs / args.steps
        cfg = {"S": S, "G": G, "P": P, "b_g": 4}
        row = {"P": P, "S": S, "G": G, "us_per_step": t * 1e6, "gb_per_s": algorithmic_bytes(cfg) / t / 1e9,
               "learner_params_per_s": S * G * P / t, "resident_bytes": h.arena_bytes,
               "l2_resident": h.arena_bytes < 126e6}
        row["frac_of_measured_peak"] = row["gb_per_s"] / peak
        rows.append(row)
        print(json.dumps(row), flush=True)
        h.close()
        del h
        torch.cuda.empty_cache()
    if args.sweep_md:
        with open(args.sweep_md, "w") as f:
            f.write(f"# Bandwidth sweep (BASELINE.json configs[4])\n\nCommand: `python bench.py --sweep --steps {args.steps} "
                    f"--warmup {args.warmup} --sweep-md {args.sweep_md}`; flat fp32, uniform gradients, diagnostics on; "
                    f"GB/s = S*P*(4G+16) / t_step; peak = {peak} GB/s ({peak_src}).  Points whose resident set is below the "
                    "126 MB L2 are marked L2: their GB/s is cache bandwidth or launch latency, not HBM.\n\n")
            f.write("| P | S | G | resident MB | us/step | GB/s | of peak | |\n|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                f.write(f"| 2^{r['P'].bit_length() - 1} | {r['S']} | {r['G']} | {r['resident_bytes'] / 1e6:.1f} | "
                        f"{r['us_per_step']:.2f} | {r['gb_per_s']:.1f} | {r['frac_of_measured_peak']:.3f} | "
                        f"{'L2' if r['l2_resident'] else ''} |\n")


def main():
    args = parse_args()
    if args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
