"""bench.py -- one JSON line per run for the H-ADPSGD super-learner step.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload swb2000] [--impl reference]

A "step" is one pass of the whole hot path (pairing, learner mean,
momentum SGD, pairwise mix, diagnostics) = ONE fused kernel launch over one batch of synthetic
gradients.  Metric (BASELINE.json): learner-params updated per second = S*G*P / t_step, with
the achieved HBM GB/s in `roofline`.  Default workload = BASELINE.json configs[2], the
145,145,344-parameter SWB-2000-shaped flat fp32 buffer with S=16 super-learners x G=4
learners (55.7 GB resident), which is the configuration the metric is quoted on.

N > 1 (torchrun), --partition:
  range (default)   ONE model of the configured size: rank r owns the parameter range
                    hadpsgd_shard_range(P, N, r) of every buffer (the method is element-wise, so there
                    is no data-path collective; only the few diagnostic doubles are all-reduced, after
                    the timed region).  Total work is fixed: "scaling": "strong".
  superlearner      the paper's topology: rank r owns S/N super-learners with all
                    P parameters; a pair whose members live on two GPUs is mixed by peer reads of the
                    partner's stage buffer inside the fused kernel (HADPSGD_PEER, CUDA IPC mappings),
                    4*P bytes per pending member per step over NVLink; steps of neighbouring ranks are
                    ordered by the library's neighbour-only epoch handshake (stream waits on the partner's
                    epoch word): no collective and no global barrier per step.  "scaling": "strong".
  weak              every rank runs its own problem of the configured size ("scaling": "weak").

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

_REAL_STDOUT = None
METRIC = "learner_params_updated_per_sec"
UNIT = "learner-params/s"
LR, MU = 0.1, 0.9
FALLBACK_HBM_GBS = 6650.0       # /opt/skills/guides/B200_PROFILING.md fallback
PCIE_GEN5_X16_GBS = 64.0        # nominal per direction; the e2e leg reports its fraction of this
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r03_traffic.csv")
KERNEL_SOURCES = ["paper_1907_05701_b200/csrc/step_kernel.cuh", "paper_1907_05701_b200/csrc/step_dispatch.cuh"]


def kernel_source_sha():
    import hashlib
    h = hashlib.sha256()
    for rel in KERNEL_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def ncu_traffic(workload, flags_text, emit):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the step kernel from the committed
    `ncu --set full` captures (profiles/r03_traffic.csv; the .md beside it names the commands).  Only a
    capture taken on THIS kernel source (sha of step_kernel.cuh + step_dispatch.cuh) for this workload
    and these flags counts; anything else is None."""
    import csv
    want = (workload, ",".join(sorted(filter(None, (t.strip() for t in flags_text.split(","))))), "1" if emit else "0")
    try:
        with open(TRAFFIC_CSV) as f:
            for row in csv.DictReader(f):
                if (row["workload"], row["flags"], row["emit_bf16"]) == want:
                    if row["kernel_source_sha16"] != kernel_source_sha():
                        return None, f"profiles/r03_traffic.csv holds a capture of another kernel source ({row['kernel_source_sha16']})"
                    return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]), \
                        f"profiles/r03_traffic.csv: {row['kernel']} at commit {row['commit']} (read {row['dram_bytes_read']} B + write {row['dram_bytes_write']} B)"
    except Exception as e:                      # no capture file: say so, never guess
        return None, f"no capture: {e}"
    return None, "no capture for this workload / flags"


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
    ap.add_argument("--cpu-sample-steps", type=int, default=10)
    ap.add_argument("--blocks-per-sm", type=int, default=0)
    ap.add_argument("--flags", default="", help="comma list: deterministic,no_diag,no_mix,eq7,share")
    ap.add_argument("--no-share-leg", action="store_true", help="skip the extra HADPSGD_SHARE_PAIR_WEIGHTS leg")
    ap.add_argument("--emit-bf16", action="store_true",
                    help="also write the bf16 working copy of the weights every step (row f2; +2 B/param)")
    ap.add_argument("--partition", default="range", choices=["range", "superlearner", "weak"],
                    help="how N > 1 GPUs share the work (ignored for N = 1)")
    ap.add_argument("--emulate-ranks", type=int, default=0,
                    help="N = 1 only: time the super-learner partition over R HADPSGD_PEER handles on ONE GPU (one stream; "
                         "peer reads are local HBM reads) -- kernel cost of the partition, not an NVLink measurement")
    ap.add_argument("--no-ceiling", action="store_true", help="skip the pure-read / pure-write membench legs (roofline.reference_mix)")
    ap.add_argument("--no-secondary", action="store_true",
                    help="skip the device-timed legs of the other kernel families (`secondary`) and the bf16 e2e leg")
    ap.add_argument("--cpu-repeats", type=int, default=3)
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE.json configs[4]: bandwidth sweep over P, S, G (one JSON line per point)")
    ap.add_argument("--sweep-md", default="", help="also write the sweep as a markdown table to this path")
    ap.add_argument("--sweep-max-log2", type=int, default=28, help="only sweep points with P <= 2^N")
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


def time_oracle(cfg, n_elems, steps, warmup=1, repeats=1, lo=0):
    """The oracle as it stands (single thread, oracle/hadpsgd_oracle.cpp) on a bounded sample:
    n_elems parameters (from `lo`) of every buffer of the workload (the method is element-wise
    independent, so a window is the same work per parameter).  Returns (seconds per step of each
    repeat, n)."""
    import numpy as np
    import oracle
    from fixtures import problem
    S, G = cfg["S"], cfg["G"]
    n = min(n_elems, cfg["P"] - lo)
    bf16 = cfg["grad"] == "bf16"
    w = problem.host_weights(7, S, lo, lo + n)
    v = np.zeros((S, n), np.float32)
    g = problem.host_grads(7, 0, S, G, lo, lo + n, cfg["dist"], bf16=bf16)
    for k in range(warmup):
        oracle.step(g, w, v, LR, MU, k, diag=True)
    times = []
    for r in range(max(repeats, 1)):
        t0 = time.perf_counter()
        for k in range(steps):
            oracle.step(g, w, v, LR, MU, warmup + k, diag=True)
        times.append((time.perf_counter() - t0) / max(steps, 1))
    return times, n


def time_oracle_all_cores(cfg, n_elems_per_thread, steps):
    """The same single-threaded oracle, one instance per hardware thread, each on its own disjoint
    element window (the C call releases the GIL).  Returns (seconds for `steps` steps, threads, n)."""
    import numpy as np
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    from fixtures import problem
    S, G = cfg["S"], cfg["G"]
    threads = os.cpu_count() or 1
    n = min(n_elems_per_thread, cfg["P"] // threads)
    bf16 = cfg["grad"] == "bf16"
    work = []
    for t in range(threads):
        lo = t * n
        work.append((problem.host_grads(7, 0, S, G, lo, lo + n, cfg["dist"], bf16=bf16),
                     problem.host_weights(7, S, lo, lo + n), np.zeros((S, n), np.float32)))

    def run(item):
        g, w, v = item
        for k in range(steps):
            oracle.step(g, w, v, LR, MU, k, diag=True)

    with ThreadPoolExecutor(max_workers=threads) as pool:
        list(pool.map(run, [(g, w.copy(), v.copy()) for g, w, v in work]))     # warm-up pass
        t0 = time.perf_counter()
        list(pool.map(run, work))
        dt = time.perf_counter() - t0
    return dt, threads, n


def cpu_baseline(cfg, n_elems, steps, repeats=3, all_cores=True):
    """`value` = the best of `repeats` repeats of the single-threaded oracle (its contract); the spread
    of the repeats is reported next to it, and -- optionally -- the same oracle run by every hardware
    thread on disjoint windows."""
    times, n = time_oracle(cfg, n_elems, steps, repeats=repeats)
    model, ncpu = host_cpu()
    per = cfg["S"] * cfg["G"] * n
    best = min(times)
    out = {"value": per / best, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"first {n} of {cfg['P']} params of every buffer (S={cfg['S']}, G={cfg['G']}), best of {len(times)} "
                     f"repeats of {steps} steps after 1 warm-up, diagnostics on; single thread; host has {ncpu} logical CPUs ({model})",
           "repeats": [per / t for t in times], "spread": (max(times) - min(times)) / min(times),
           "gb_per_s": cfg["S"] * n * (cfg["G"] * cfg["b_g"] + 16) / best / 1e9,
           "ms_per_step_sample": best * 1e3}
    if all_cores:
        dt, threads, m = time_oracle_all_cores(cfg, 1 << 18, 5)
        out["all_cores"] = {"value": cfg["S"] * cfg["G"] * m * threads * 5 / dt, "unit": UNIT, "cores": threads,
                            "sample": f"{threads} threads, each the single-threaded oracle on its own {m}-param window, 5 steps"}
    return out


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = workload(args.workload)
    times, n = time_oracle(cfg, args.cpu_sample_elems, args.steps, warmup=min(args.warmup, 2))
    dt = times[0]
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
    # what the link itself delivers on this box: the same pinned buffers copied to the gradient region with
    # nothing else running (outside the timed region; the gradients on the device are left as they were)
    link = None
    if world == 1:
        pairs = [(h.hadpsgd_grads(b // G if n_host == S * G else 0, b % G).view(torch.uint8), host[b]) for b in range(min(n_host, 8))]
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for dst, src in pairs:
            dst.copy_(src, non_blocking=True)
        torch.cuda.synchronize()
        link = len(pairs) * nbytes / (time.perf_counter() - t0) / 1e9
    note = f"{n_host} distinct pinned host buffers of {nbytes} B"
    return max(dev, wall), S * G * nbytes, 3 * S * 8, note, link


def make_problem(H, torch, dist, args, cfg, flags, local, rank, world):
    """Builds this rank's handle for the chosen partition and fills it.  Returns (handle, info)."""
    from fixtures import device, generator as gen, problem
    S, G, P = cfg["S"], cfg["G"], cfg["P"]
    gdt = H.BF16 if cfg["grad"] == "bf16" else H.F32
    wdt = H.BF16 if args.emit_bf16 else H.F32
    # N = 1: one plain handle, unless launched by torch.distributed.run with an explicit partition (a
    # one-rank smoke test of the partition's plumbing)
    part = args.partition if (world > 1 or (dist is not None and args.partition == "superlearner")) else "single"
    dist_name = cfg["dist"]
    if part in ("single", "weak"):
        h = H.Hadpsgd(S, G, cfg["seg_len"], gdt, flags, device=local, working_dtype=wdt)
        seed = 2000 + rank            # weak: every rank is its own problem
        problem.fill_weights(h, seed)
        problem.fill_grads(h, seed, 0, dist_name)
        info = {"units": S * G * P, "scaling": "weak", "partition": part,
                "parallelism": "single GPU" if world == 1 else f"weak: {world} independent problems of the configured size, no collective"}
        return h, info
    if part == "range":
        # ONE model: rank r owns the element range [lo, hi) of every buffer (hadpsgd_shard_range)
        lay = H.hadpsgd_layout(S, G, cfg["seg_len"], gdt, wdt)
        assert lay["P_padded"] == P, "--partition range needs a segment table without padding (all BLSTM tables are)"
        lo, hi = H.hadpsgd_shard_range(P, world, rank)
        h = H.Hadpsgd(S, G, [hi - lo], gdt, flags, device=local, working_dtype=wdt)
        seed = 2000
        for s_ in range(S):
            device.fill(h.hadpsgd_weights(s_)[:hi - lo], gen.stream_key(seed, gen.STREAM_WEIGHT, 0, s_, 0), "normal", 0.05,
                        elem_offset=lo)
            for g_ in range(G):
                device.fill(h.hadpsgd_grads(s_, g_)[:hi - lo], gen.stream_key(seed, gen.STREAM_GRAD, 0, s_, g_), dist_name, 1e-3,
                            elem_offset=lo)
        info = {"units": S * G * (hi - lo), "scaling": "strong", "shard": [lo, hi], "partition": part,
                "parallelism": f"range: one {P}-parameter model, rank r owns hadpsgd_shard_range(P, {world}, r) of every buffer; "
                               "no data-path collective (diagnostics all-reduced after the timed region)"}
        return h, info
    # superlearner: rank r owns S/world super-learners with all P parameters
    assert S % world == 0, "--partition superlearner needs S divisible by the number of GPUs"
    assert not args.emit_bf16 and not (flags & (H.SHARE_PAIR_WEIGHTS | H.EQ7_LITERAL)), "peer mode: no emit / share / eq7"
    S_l = S // world
    rank_begin = [r * S_l for r in range(world + 1)]
    h = H.Hadpsgd(S_l, G, cfg["seg_len"], gdt, flags | H.PEER, device=local, own_arena=True)
    h.hadpsgd_peer_init(rank, world, rank_begin)
    ipc, off = h.hadpsgd_peer_ipc_export()
    mine = torch.tensor(list(ipc) + list(off.to_bytes(8, "little")), dtype=torch.uint8, device="cuda")
    got = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(got, mine)
    for r in range(world):
        if r != rank:
            raw = bytes(got[r].cpu().tolist())
            h.hadpsgd_peer_ipc_attach(r, raw[:64], int.from_bytes(raw[64:], "little"))
    seed = 2000
    nat = problem.natural_offsets(h.seg_len)
    for s_ in range(S_l):
        sg = rank_begin[rank] + s_
        for k_, n_ in enumerate(h.seg_len):
            o_, _ = h.hadpsgd_segment(k_)
            device.fill(h.hadpsgd_weights(s_)[o_:o_ + n_], gen.stream_key(seed, gen.STREAM_WEIGHT, 0, sg, 0), "normal", 0.05,
                        elem_offset=int(nat[k_]))
            for g_ in range(G):
                device.fill(h.hadpsgd_grads(s_, g_)[o_:o_ + n_], gen.stream_key(seed, gen.STREAM_GRAD, 0, sg, g_), dist_name, 1e-3,
                            elem_offset=int(nat[k_]))
    # expected NVLink traffic: every member whose ring partner lives on another GPU publishes u on the
    # odd (or even) step and reads its partner's 4*P bytes at the next launch
    strad = [sum(1 for sg in range(rank_begin[rank], rank_begin[rank + 1])
                 if not rank_begin[rank] <= H.hadpsgd_pairing(S, k)[sg] < rank_begin[rank + 1]) for k in (0, 1)]
    info = {"units": S_l * G * P, "scaling": "strong", "barrier": True, "partition": part,
            "nvlink_read_bytes_per_rank_per_step": [strad[1] * 4 * P, strad[0] * 4 * P],   # [even step reads what the odd step left, odd step ...]
            "parallelism": f"superlearner: rank r owns super-learners [{S_l}r, {S_l}(r+1)) of {S}; straddling pairs mixed by peer reads "
                           f"of the partner's stage buffer inside the fused kernel (CUDA IPC); no per-step collective: the library's neighbour-only "
                           f"epoch handshake (stream waits on the partners' epoch words) orders the ranks"}
    return h, info


def time_device_steps_barrier(torch, dist, h, steps, warmup, k0=0, sampler=None):
    """As time_device_steps, for --partition superlearner.  Nothing is enqueued between the steps: the ranks
    are ordered by the library's neighbour-only epoch handshake.  One NCCL all-reduce runs in the warm-up
    (outside the timed region) so that a multi-GPU run still shows its communicator in NCCL_DEBUG output."""
    tok = torch.zeros(1, device="cuda")
    dist.all_reduce(tok)
    for k in range(warmup):
        h.hadpsgd_step(LR, MU, k0 + k)
    torch.cuda.synchronize()
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
    dist.barrier()
    torch.cuda.synchronize()
    return ev0.elapsed_time(ev1) / 1e3, clocks


def reference_mix_rate(torch, read_bytes, write_bytes):
    """This box's pure-read and pure-write streaming rates (fixtures/membench.cu, the step kernel's access
    shape) and the rate they imply for this kernel's byte mix if reads and writes simply took turns on the
    DRAM bus: t = read_bytes / BW_read + write_bytes / BW_write.  A REFERENCE rate, not an upper bound: the
    membench legs are one plain kernel each (one block per SM) and the step kernel has measured up to 3 %
    above the figure, so a fraction slightly over 1 is not an inconsistency."""
    from fixtures import device
    r = device.membench(8 << 30, 12, write=False, reps=3)
    w = device.membench(8 << 30, 4, write=True, reps=3)
    t = read_bytes / (r * 1e9) + write_bytes / (w * 1e9)
    return {"read_gbs": r, "write_gbs": w, "mix_gbs": (read_bytes + write_bytes) / t / 1e9,
            "how": "fixtures/membench.cu: 12 read streams / 4 write streams, 32 B accesses, 148 x 256 threads, best of 3; "
                   "mix = bytes / (read_bytes / read_gbs + write_bytes / write_gbs); a reference rate for this byte mix, "
                   "not an upper bound (the legs are untuned single kernels)"}


def secondary_leg(H, torch, args, name, emit):
    """One more kernel family, device-timed like the headline: BASELINE.json configs[3] (ragged bf16, 8 x 8),
    the headline shape with the bf16 working copy (row f2), the paper-literal model (8 x 8 fp32)."""
    from fixtures import problem
    cfg = workload(name)
    cfg["emit"] = emit
    h = H.Hadpsgd(cfg["S"], cfg["G"], cfg["seg_len"], H.BF16 if cfg["grad"] == "bf16" else H.F32, 0, device=0,
                  working_dtype=H.BF16 if emit else H.F32)
    problem.fill_weights(h, 2000)
    problem.fill_grads(h, 2000, 0, cfg["dist"])
    torch.cuda.synchronize()
    n0 = h.hadpsgd_launch_count()
    secs, clocks = time_device_steps(torch, None, h, args.steps, args.warmup, sampler=ClockSampler(0))
    launches = h.hadpsgd_launch_count() - n0 - args.warmup
    t = secs / args.steps
    abytes = cfg["S"] * h.P_padded * (cfg["G"] * cfg["b_g"] + 16 + (2 if emit else 0))
    traffic, src = ncu_traffic(name, "", emit)
    h.close()
    del h
    torch.cuda.empty_cache()
    return {"workload": name, "working_dtype": "bf16" if emit else "f32", "S": cfg["S"], "G": cfg["G"], "P": cfg["P"],
            "grad_dtype": cfg["grad"], "ms_per_step": t * 1e3, "value": cfg["S"] * cfg["G"] * cfg["P"] / t, "unit": UNIT,
            "algorithmic_bytes_per_launch": abytes, "achieved_gbs": abytes / t / 1e9,
            "frac_of_8TBps_nominal": abytes / t / 1e9 / 8000.0, "frac_of_measured_copy_peak": abytes / t / 1e9 / measured_peak()[0],
            "traffic": traffic, "traffic_source": src, "gpu_launches": launches, "steps": args.steps, "warmup": args.warmup,
            "clocks": clocks}


def e2e_leg_bf16(H, torch, args):
    """The end-to-end call (hadpsgd_step_host, pinned host gradients, copies inside the timed region) on the
    bf16-gradient handle of configs[3]: half the PCIe bytes per learner-parameter of the fp32 headline."""
    from fixtures import problem
    cfg = workload("swb2000_ragged_bf16")
    h = H.Hadpsgd(cfg["S"], cfg["G"], cfg["seg_len"], H.BF16, 0, device=0)
    problem.fill_weights(h, 2000)
    problem.fill_grads(h, 2000, 0, cfg["dist"])
    torch.cuda.synchronize()
    secs, h2d, d2h, note, link = time_e2e_steps(torch, None, h, cfg, args.e2e_steps)
    h.close()
    del h
    torch.cuda.empty_cache()
    e_step = secs / args.e2e_steps
    return {"workload": "swb2000_ragged_bf16", "value": cfg["S"] * cfg["G"] * cfg["P"] / e_step, "unit": UNIT,
            "ms_per_step": e_step * 1e3, "steps": args.e2e_steps, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
            "h2d_gbs": h2d / e_step / 1e9, "link_gbs_plain_copy": link, "note": "hadpsgd_step_host on bf16 gradients: " + note}


def run_ours(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback (use --impl reference for the oracle)")
    import paper_1907_05701_b200 as H
    H.lib()                                   # fail loudly if libhadpsgd.so is missing

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    # The oracle baseline first, in a process that has not touched CUDA yet: with a CUDA context and tens
    # of GB of pinned host memory mapped, the same single-threaded oracle runs 1.6 x slower (its 268 MB
    # scratch vector is allocated and faulted in every step) -- measured as it stands either way, but the
    # clean process is the fairer baseline and is what --impl reference sees too.
    cpu_line = None
    if world == 1 and rank == 0 and not args.no_cpu_baseline:
        cpu_line = cpu_baseline(workload(args.workload), args.cpu_sample_elems, args.cpu_sample_steps, args.cpu_repeats)
    dist = None
    if world > 1 or "RANK" in os.environ:          # launched by torch.distributed.run (any N)
        # stdout carries the one JSON line only: NCCL prints its version banner to fd 1, so fd 1 is
        # pointed at stderr for the rest of the run and the line goes out through a saved copy
        global _REAL_STDOUT
        sys.stdout.flush()
        _REAL_STDOUT = os.fdopen(os.dup(1), "w")
        os.dup2(2, 1)
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    assert world == args.gpus, f"--gpus {args.gpus} but WORLD_SIZE={world} (launch N>1 with torch.distributed.run)"

    cfg = workload(args.workload)
    cfg["emit"] = args.emit_bf16
    S, G, P = cfg["S"], cfg["G"], cfg["P"]
    flags = parse_flags(H, args.flags)
    h, info = make_problem(H, torch, dist, args, cfg, flags, local, rank, world)
    if args.blocks_per_sm:
        h.hadpsgd_set_launch(args.blocks_per_sm)
    torch.cuda.synchronize()
    timer = time_device_steps_barrier if info.get("barrier") else time_device_steps

    n0 = h.hadpsgd_launch_count()
    secs, clocks = timer(torch, dist, h, args.steps, args.warmup, sampler=ClockSampler(local) if rank == 0 else None)
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
        secs, clocks = timer(torch, dist, h, args.steps, args.warmup, k0=args.steps + args.warmup,
                             sampler=ClockSampler(local) if rank == 0 else None)
        launches = h.hadpsgd_launch_count() - n0 - args.warmup
    if clocks is not None:
        clocks["remeasured_after_slowdown"] = remeasured
    diag = None if (flags & H.NO_DIAG) else h.hadpsgd_diagnostics()

    e2e = None
    if not args.no_e2e and not info.get("barrier"):
        e2e = time_e2e_steps(torch, dist, h, cfg, args.e2e_steps)   # (seconds, h2d bytes, d2h bytes, note, plain link GB/s)

    # max over ranks (device time), units and diagnostics summed over the ranks
    units = info["units"]
    if dist is not None:
        from paper_1907_05701_b200 import sharding
        secs = sharding.max_over_ranks(secs, dist, "cuda")
        t_units = torch.tensor([float(units)], dtype=torch.float64, device="cuda")
        dist.all_reduce(t_units)
        units = float(t_units[0])
        if e2e:
            e2e = (sharding.max_over_ranks(e2e[0], dist, "cuda"),) + e2e[1:]
        if diag is not None and info.get("partition") == "range":
            # the only collective of the range partition: 3*S doubles, outside the timed region
            diag = sharding.allreduce_diagnostics(diag, dist, "cuda")
    arena_bytes = h.arena_bytes
    P_rank = h.P_padded
    S_rank = h.S
    h.close()
    del h
    torch.cuda.empty_cache()

    # Second device-timed leg, reported beside the headline (never instead of it): the same step with
    # HADPSGD_SHARE_PAIR_WEIGHTS, where pair members share one weight buffer (same arithmetic and
    # results; one weight write per pair and one HBM fetch of the buffer two pairs read).
    shared = None
    can_share = (not (flags & (H.NO_MIX | H.EQ7_LITERAL | H.SHARE_PAIR_WEIGHTS)) and S > 1 and S % 2 == 0
                 and info.get("partition") in ("single", "weak"))
    if can_share and not args.no_share_leg:
        from fixtures import problem
        hs = H.Hadpsgd(S, G, cfg["seg_len"], H.BF16 if cfg["grad"] == "bf16" else H.F32, flags | H.SHARE_PAIR_WEIGHTS,
                       device=local, working_dtype=H.BF16 if args.emit_bf16 else H.F32)
        problem.fill_weights(hs, 2000 + rank)
        problem.fill_grads(hs, 2000 + rank, 0, cfg["dist"])
        torch.cuda.synchronize()
        s_secs, _ = time_device_steps(torch, dist, hs, args.steps, args.warmup)
        if dist is not None:
            from paper_1907_05701_b200 import sharding
            s_secs = sharding.max_over_ranks(s_secs, dist, "cuda")
        shared = s_secs / args.steps
        hs.close()
        del hs
        torch.cuda.empty_cache()

    # Device-timed legs of the other kernel families, beside the headline (never instead of it): same
    # steps / warm-up, each with its own clock record.  Only on the default single-GPU headline run.
    secondary = None
    e2e_bf16 = None
    if (world == 1 and dist is None and not args.no_secondary and args.workload == "swb2000" and not args.flags
            and not args.emit_bf16 and not args.blocks_per_sm):
        secondary = [secondary_leg(H, torch, args, name, emit) for name, emit in
                     (("swb2000_ragged_bf16", False), ("swb2000", True), ("paper_literal", False))]
        if not args.no_e2e:
            e2e_bf16 = e2e_leg_bf16(H, torch, args)

    if rank == 0:
        t_step = secs / args.steps
        peak, peak_src = measured_peak()
        per_sp = cfg["G"] * cfg["b_g"] + 16 + (2 if cfg.get("emit") else 0)        # bytes per super-learner-parameter
        abytes_rank = S_rank * P_rank * per_sp                                      # algorithmic bytes of ONE launch (this rank)
        achieved = abytes_rank / t_step / 1e9
        traffic, traffic_src = (None, "n/a: per-rank launch of a partition") if info.get("partition") != "single" else \
            ncu_traffic(args.workload, args.flags, args.emit_bf16)
        roof = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": abytes_rank,
                "kernel": "hadpsgd::step_kernel (one launch = one step)", "frac_of_8TBps_nominal": achieved / 8000.0,
                "note": "peak is a 1:1 copy; this kernel reads more than it writes, and reads are the faster direction, "
                        "so frac may exceed 1 (see reference_mix)"}
        if "nvlink_read_bytes_per_rank_per_step" in info:
            # fused compute + peer-read kernel: the floor of a step is the slower of its local HBM bytes at the
            # measured HBM peak and its NVLink bytes at the measured peer-copy rate (B200_PROFILING.md: 770 GB/s)
            nv = info["nvlink_read_bytes_per_rank_per_step"]
            floors = [max(abytes_rank / (peak * 1e9), b / 770e9) for b in nv]
            roof["nvlink"] = {"read_bytes_per_rank": {"even_step": nv[0], "odd_step": nv[1]}, "peer_gbs_reference": 770.0,
                              "floor_ms_even_odd": [f * 1e3 for f in floors],
                              "frac_of_floor": (sum(floors) / len(floors)) / t_step,
                              "note": "floor = max(local bytes / measured HBM peak, peer bytes / 770 GB/s) per step parity"}
        if not args.no_ceiling and world == 1:
            rd = S_rank * P_rank * (cfg["G"] * cfg["b_g"] + 8)
            ref = reference_mix_rate(torch, rd, abytes_rank - rd)
            ref["frac_of_reference_mix_rate"] = achieved / ref["mix_gbs"]
            roof["reference_mix"] = ref
        line = {
            "metric": METRIC, "value": units / t_step, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_step * 1e3, "higher_is_better": True,
            "scaling": info["scaling"], "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "S": S, "G": G, "P": P, "n_segments": len(cfg["seg_len"]),
                       "grad_dtype": cfg["grad"], "master_dtype": "f32",
                       "working_dtype": "bf16" if args.emit_bf16 else "f32", "lr": LR, "momentum": MU,
                       "resident_bytes_per_gpu": arena_bytes, "flags": args.flags or "default (diagnostics on)",
                       "l2": "inputs larger than L2 (working set per step >> 126 MB); no flush needed",
                       "partition": info.get("partition", "single"), "parallelism": info["parallelism"]},
            "roofline": roof, "clocks": clocks, "gpu_launches": launches,
        }
        for k_ in ("shard", "nvlink_read_bytes_per_rank_per_step"):
            if k_ in info:
                line["config"][k_] = info[k_]
        if diag is not None:
            line["diagnostics_last_step"] = {"gsq_sum": float(diag["gsq"].sum()), "wsq_sum": float(diag["wsq"].sum()),
                                             "gap_sum": float(diag["gap"].sum())}
        if shared is not None:
            abytes = S * P * per_sp
            line["share_pair_weights"] = {
                "flag": "HADPSGD_SHARE_PAIR_WEIGHTS (opt-in; bench.py --flags share makes it the headline leg)",
                "ms_per_step": shared * 1e3, "value": world * S * G * P / shared, "unit": UNIT,
                "achieved_algorithmic_gbs": abytes / shared / 1e9, "frac_of_peak_algorithmic": abytes / shared / 1e9 / peak,
                "bytes_moved_model": S * P * (cfg["G"] * cfg["b_g"] + 12 + (1 if args.emit_bf16 else 0)),
                "traffic": ncu_traffic(args.workload, ",".join(filter(None, [args.flags, "share"])), args.emit_bf16)[0],
                "note": "same arithmetic and results (parity-tested at full size); pair members share one of the S weight "
                        "buffers: 4 B less written and 4 B less fetched from HBM per pair-parameter than the algorithmic "
                        "S*P*(G*b_g+16), so achieved_algorithmic_gbs exceeds the DRAM rate actually sustained"}
        if e2e:
            e_step = e2e[0] / args.e2e_steps
            h2d_gbs = e2e[1] / e_step / 1e9
            line["e2e"] = {"value": units / e_step, "unit": UNIT, "h2d_bytes_per_step": e2e[1],
                           "d2h_bytes_per_step": e2e[2], "ms_per_step": e_step * 1e3, "steps": args.e2e_steps,
                           "h2d_gbs": h2d_gbs, "frac_of_pcie_gen5_x16": h2d_gbs / PCIE_GEN5_X16_GBS,
                           "link_gbs_plain_copy": e2e[4], "frac_of_plain_copy": (h2d_gbs / e2e[4]) if e2e[4] else None,
                           "note": "hadpsgd_step_host: " + e2e[3] + "; bound by the host-to-device copy of the S*G gradient "
                                   f"buffers (PCIe Gen5 x16, {PCIE_GEN5_X16_GBS:.0f} GB/s nominal per direction), which the "
                                   "fused kernel overlaps chunk by chunk; the new weights and momenta stay resident in HBM "
                                   "(the learners live on the GPU), so the device-to-host traffic is the diagnostics only"}
        if secondary is not None:
            line["secondary"] = secondary
        if e2e_bf16 is not None:
            line["e2e_bf16"] = e2e_bf16
        if cpu_line is not None:
            line["cpu_baseline"] = cpu_line
        print(json.dumps(line), file=_REAL_STDOUT or sys.stdout, flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_emulated_partition(args):
    """--emulate-ranks R: the super-learner partition of the workload over R PEER handles on
    one GPU and one stream.  A step = the step of every handle.  Even and odd ring steps differ (odd steps
    publish u, even steps resolve the pending mixes), so they are timed separately; `value` uses their mean."""
    import torch
    import paper_1907_05701_b200 as H
    from fixtures import device, generator as gen
    H.lib()
    torch.cuda.set_device(0)
    cfg = workload(args.workload)
    S, G, P, R = cfg["S"], cfg["G"], cfg["P"], args.emulate_ranks
    assert S % R == 0 and len(cfg["seg_len"]) == 1, "--emulate-ranks needs S divisible by R and a flat workload"
    S_l = S // R
    rb = [r * S_l for r in range(R + 1)]
    gdt = H.BF16 if cfg["grad"] == "bf16" else H.F32
    hs = [H.Hadpsgd(S_l, G, cfg["seg_len"], gdt, parse_flags(H, args.flags) | H.PEER, device=0) for _ in range(R)]
    for r, h in enumerate(hs):
        h.hadpsgd_peer_init(r, R, rb)
    for r, h in enumerate(hs):
        for q, other in enumerate(hs):
            if q != r:
                h.hadpsgd_peer_attach(q, other.hadpsgd_peer_stage())
        for s_ in range(S_l):
            device.fill(h.hadpsgd_weights(s_), gen.stream_key(2000, gen.STREAM_WEIGHT, 0, rb[r] + s_, 0), "normal", 0.05)
            for g_ in range(G):
                device.fill(h.hadpsgd_grads(s_, g_), gen.stream_key(2000, gen.STREAM_GRAD, 0, rb[r] + s_, g_), cfg["dist"], 1e-3)
    torch.cuda.synchronize()
    k = 0
    for _ in range(max(args.warmup, 3) // 2 * 2 + 2):
        for h in hs:
            h.hadpsgd_step(LR, MU, k)
        k += 1
    torch.cuda.synchronize()
    n0 = sum(h.hadpsgd_launch_count() for h in hs)
    sampler = ClockSampler(0)
    sampler.start()
    per = {0: [], 1: []}
    for _ in range(args.steps):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for h in hs:
            h.hadpsgd_step(LR, MU, k)
        ev1.record()
        torch.cuda.synchronize()
        per[k % 2].append(ev0.elapsed_time(ev1) / 1e3)
        k += 1
    clocks = sampler.stop()
    launches = sum(h.hadpsgd_launch_count() for h in hs) - n0
    even, odd = sum(per[0]) / max(len(per[0]), 1), sum(per[1]) / max(len(per[1]), 1)
    t_step = (sum(per[0]) + sum(per[1])) / args.steps
    pending_even = sum(1 for sg in range(S) if H.hadpsgd_pairing(S, 1)[sg] // S_l != sg // S_l)   # left pending by odd steps
    abytes = algorithmic_bytes(cfg)
    peak, peak_src = measured_peak()
    for h in hs:
        h.close()
    line = {"metric": METRIC, "value": S * G * P / t_step, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_step * 1e3, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": args.workload, "S": S, "G": G, "P": P, "partition": "superlearner (emulated)", "emulated_ranks": R,
                       "parallelism": f"{R} HADPSGD_PEER handles ({S_l} super-learners each) on ONE GPU and one stream: the kernels of "
                                      "the partition with peer reads served from local HBM; NOT an NVLink measurement",
                       "ms_even_step": even * 1e3, "ms_odd_step": odd * 1e3,
                       "stage_bytes_read_per_even_step": pending_even * 4 * P,
                       "note": "odd ring steps: straddling members publish u (same bytes as a plain step); even steps: every pending "
                               "member also reads its partner's stage buffer (4 B per parameter on top of the algorithmic bytes)"},
            "roofline": {"bound": "hbm", "achieved": abytes / t_step / 1e9, "peak": peak, "unit": "GB/s",
                         "frac": abytes / t_step / 1e9 / peak, "traffic": None, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": abytes, "frac_of_8TBps_nominal": abytes / t_step / 1e9 / 8000.0,
                         "achieved_even_step_incl_stage_reads": (abytes + pending_even * 4 * P) / even / 1e9 if even else None},
            "clocks": clocks, "gpu_launches": launches}
    print(json.dumps(line), flush=True)


def run_sweep(args):
    """BASELINE.json configs[4]: flat fp32 buffer of 2^10..2^28 params (powers of 4), G in {2,4,8},
    S in {2,4,8,16} with S*G*P*4 B <= 96 GB; uniform grads in [-1e-3, 1e-3]; W warm + K timed steps
    per point (defaults 5 + 20); GB/s (algorithmic) vs buffer size.  Every point is timed twice: the K
    steps enqueued one by one from Python ("eager": below ~10 us per step this measures the host's launch
    path, not the GPU), and the same K steps captured once into a CUDA graph and replayed (what a
    launch-bound caller does; hadpsgd_step only enqueues, so it captures).  Small points are L2-resident
    (working set < 126 MB) and latency-bound: they are flagged, not bandwidth claims."""
    import torch
    import paper_1907_05701_b200 as H
    from fixtures import problem, shapes
    H.lib()
    torch.cuda.set_device(0)
    peak, peak_src = measured_peak()
    side = torch.cuda.Stream()
    rows = []
    for P, S, G in shapes.sweep_points():
        if P > (1 << args.sweep_max_log2):
            continue
        with torch.cuda.stream(side):
            h = H.Hadpsgd(S, G, [P], H.F32, parse_flags(H, args.flags), device=0, stream=side)
            problem.fill_weights(h, 3000)
            problem.fill_grads(h, 3000, 0, "uniform")
            torch.cuda.synchronize()
            secs, _ = time_device_steps(torch, None, h, args.steps, args.warmup)
            t_eager = secs / args.steps
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                for k in range(args.steps):
                    h.hadpsgd_step(LR, MU, k)
            for _ in range(max(1, args.warmup // 2)):
                graph.replay()
            torch.cuda.synchronize()
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev0.record(side)
            graph.replay()
            ev1.record(side)
            torch.cuda.synchronize()
            t_graph = ev0.elapsed_time(ev1) / 1e3 / args.steps
        t = min(t_eager, t_graph)
        cfg = {"S": S, "G": G, "P": P, "b_g": 4}
        row = {"P": P, "S": S, "G": G, "us_per_step": t * 1e6, "us_per_step_eager": t_eager * 1e6,
               "us_per_step_graph": t_graph * 1e6, "gb_per_s": algorithmic_bytes(cfg) / t / 1e9,
               "learner_params_per_s": S * G * P / t, "resident_bytes": h.arena_bytes,
               "l2_resident": h.arena_bytes < 126e6,
               # a step that moves < 2 GiB keeps the last 64 MB it stores in L2 for the next step (serpentine walk)
               "l2_assisted": algorithmic_bytes(cfg) < (2 << 30)}
        row["frac_of_measured_peak"] = row["gb_per_s"] / peak
        rows.append(row)
        print(json.dumps(row), flush=True)
        h.close()
        del h, graph
        torch.cuda.empty_cache()
    if args.sweep_md:
        with open(args.sweep_md, "w") as f:
            diag_txt = "diagnostics OFF (`--flags no_diag`; the same kernels a handle runs after `hadpsgd_set_diagnostics(h, 0)`)" \
                if "no_diag" in args.flags else "diagnostics on"
            flag_txt = f" --flags {args.flags}" if args.flags else ""
            f.write(f"# Bandwidth sweep (BASELINE.json configs[4])\n\nCommand: `python bench.py --sweep --steps {args.steps} "
                    f"--warmup {args.warmup}{flag_txt} --sweep-md {args.sweep_md}`; flat fp32, uniform gradients, {diag_txt}; "
                    f"each point: {args.steps} steps enqueued from Python (eager) and the same {args.steps} steps as one CUDA-graph "
                    f"replay; us/step = the faster of the two; GB/s = S*P*(4G+16) / t_step (ALGORITHMIC bytes per second); "
                    f"peak = {peak} GB/s ({peak_src}).  "
                    "`L2`: the resident set is below the 126 MB L2 -- cache bandwidth or launch latency, not HBM.  `L2 part`: a step "
                    "moves less than 2 GiB, so the serpentine walk (DESIGN.md section 6) serves part of it from L2 -- the step before "
                    "left its last 64 MB of stores there -- and GB/s can exceed what HBM delivers.  Unmarked points are HBM-bound.\n\n")
            f.write("| P | S | G | resident MB | us/step eager | us/step graph | GB/s | of peak | |\n|---|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                f.write(f"| 2^{r['P'].bit_length() - 1} | {r['S']} | {r['G']} | {r['resident_bytes'] / 1e6:.1f} | "
                        f"{r['us_per_step_eager']:.2f} | {r['us_per_step_graph']:.2f} | {r['gb_per_s']:.1f} | "
                        f"{r['frac_of_measured_peak']:.3f} | {'L2' if r['l2_resident'] else 'L2 part' if r['l2_assisted'] else ''} |\n")


def main():
    args = parse_args()
    if args.sweep:
        run_sweep(args)
    elif args.emulate_ranks and args.impl == "ours":
        run_emulated_partition(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
