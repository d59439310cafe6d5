#!/usr/bin/env python
"""bench.py -- the benchmark contract for the AES-CTR offload engine.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--backend engine|launch] [--workload c2|c3] [--no-extras] [--sweep [--sweep-out F]]

A *step* is one pass of the whole hot path (submit -> dispatch -> counter
blocks -> cipher -> XOR/store -> completion) over one batch of synthetic input.  At N = 1 the batch
is BASELINE.json configs[1], the configuration the metric is quoted on: 1,000 requests of 1 MiB,
AES-128-CTR, one shared key, distinct nonces, 64 in flight (closed loop: the next request is
submitted when one completes), payloads resident in HBM.  `value` is payload GB/s of the whole job.

--backend engine (default) is the product path: the persistent kernel fed by the host-mapped ring.
  aes_engine_start (step a0: the one kernel launch the engine ever makes) happens once, right before
  the timed region  [sync, barrier | K steps | events, sync]; its cost is reported as engine_start_ms.
--sweep prints BASELINE.json configs[4] (size x in-flight x key size) instead, one JSON line per cell.
--backend launch runs the same worker code through ordinary launches (aes_ctr_launch_batch, 64
  requests per launch: the paper's own "stream + event" mechanism).  This is the form ncu can
  replay, so the committed profiles are made with it; a persistent kernel that waits for host
  submissions would deadlock under a serialising profiler.

The JSON line also carries: roofline (binding unit = the shared-memory lookup crossbar, see
DESIGN.md section 6; HBM fraction beside it), e2e (payloads in pinned HOST memory, read and written
over PCIe inside the timed region), cpu_baseline (the oracle on the host cores, bounded sample),
latency at 4 KiB (p50/p99 submit -> completion observed), clocks sampled during the timed region.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2607_02630_b200 import workloads  # noqa: E402

MIB = 1 << 20
METRIC = "aes_ctr_payload_throughput"
UNIT = "GB/s"

# shared-memory lookups per 16-byte block in the CUDA path: per block
# 1 (round 1) + 4 (round 2) + 16 * (Nr - 2); plus, per pair of consecutive rows (16 blocks per lane),
# 27 for the first row's constants and 10 for stepping them to the second row
SETUP = (27 + 10) / 16.0
LOOKUPS = {128: 1 + 4 + 16 * 8 + SETUP, 192: 1 + 4 + 16 * 10 + SETUP, 256: 1 + 4 + 16 * 12 + SETUP}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the launch backend, from the committed ncu --set full capture
# (profiles/r2_traffic.json, written from the .ncu-rep by the command named in profiles/r2_ncu.md; a persistent launch
# cannot be replayed by ncu)
def _ncu_traffic(workload):
    p = os.path.join(ROOT, "profiles", "r2_traffic.json")
    if not os.path.exists(p):
        return None, "no committed capture (profiles/r2_traffic.json)"
    d = json.load(open(p)).get(workload)
    if not d:
        return None, "no capture for %s in profiles/r2_traffic.json" % workload
    return float(d["dram_bytes_read"]) + float(d["dram_bytes_write"]), d.get("how", "profiles/r2_traffic.json")


SMEM_BYTES_PER_CLK_PER_SM = 128.0  # 32 banks x 4 B (guides/B300_MICROARCH.md "smem crossbar BW")


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


# --------------------------------------------------------------------------------------------
# clocks sampled DURING the timed region (NVML; the timed calls release the GIL)
# --------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index: int):
        self.samples, self.power, self.reasons = [], [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._th = None
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:  # noqa: BLE001
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:  # noqa: BLE001
                pass
            time.sleep(0.002)

    def __enter__(self):
        if self.nv:
            self._th = threading.Thread(target=self._run, daemon=True)
            self._th.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._th:
            self._th.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "power_w_max": max(self.power) if self.power else None}


# --------------------------------------------------------------------------------------------
# workload set-up
# --------------------------------------------------------------------------------------------
def make_workload(name: str):
    if name == "c2":
        return workloads.config2(), 128
    if name == "c3":
        return workloads.config3(), 256
    raise SystemExit("unknown workload %s" % name)


def fill_payloads(w, dst_view_of):
    """Writes the seeded payload of every request through dst_view_of(i) -> writable uint8 ndarray."""
    for i in range(w.n):
        dst_view_of(i)[:] = w.payload(i)


def percentile(a, q):
    return float(np.percentile(a, q)) if len(a) else None


# --------------------------------------------------------------------------------------------
# reference arm: the oracle on the host cores
# --------------------------------------------------------------------------------------------
def oracle_sample(w, n_req):
    """The first n_req requests of w as one (n_req, size) array: built once, used by every timed pass."""
    n_req = min(n_req, w.n)
    size = int(w.length[0])
    src = np.empty((n_req, size), dtype=np.uint8)
    for i in range(n_req):
        src[i] = w.payload(i)
    return src


def oracle_throughput(w, keybits, n_req, cores, src=None):
    """Runs the oracle, as it stands, over the first n_req requests of w on `cores` threads.
    Returns (GB/s, seconds)."""
    import concurrent.futures as cf

    from oracle import oracle as o

    n_req = min(n_req, w.n)
    size = int(w.length[0])
    if src is None:
        src = oracle_sample(w, n_req)
    dst = np.empty((n_req, size), dtype=np.uint8)
    o.lib()

    def one(i):
        o.ctr_into(w.key_of(i), w.icb_of(i), src[i].ctypes.data, dst[i].ctypes.data, size)

    t0 = time.perf_counter()
    with cf.ThreadPoolExecutor(cores) as ex:
        list(ex.map(one, range(n_req)))
    dt = time.perf_counter() - t0
    return n_req * size / dt / 1e9, dt


def oracle_requests_per_pass(w, keybits, cores, passes, budget_s=150.0):
    """How much of the workload one timed pass of the oracle covers: ALL of it ("configs 2 and 3 in
    full") when `passes` such passes fit about budget_s seconds at the rate a short probe measures on this box, else the
    largest prefix that does, never less than one request per core.  Both arms of bench.py size their sample here."""
    probe = max(cores, 8)
    gbs, _ = oracle_throughput(w, keybits, probe, cores)
    fit = int(budget_s * gbs * 1e9 / max(passes, 1) / int(w.length[0]))
    return int(min(w.n, max(cores, fit)))


def verify_against_oracle(jobs, window=MIB):
    """jobs: (key, icb, plaintext uint8 ndarray, output uint8 ndarray).  Every byte of every job against the oracle,
    in windows of `window` bytes (oracle_ctr_at: counter = ICB + offset / 16) spread over the host cores.
    Returns (bytes verified, number of windows that differ).  Test infrastructure: runs after the timed regions."""
    import concurrent.futures as cf

    from oracle import oracle as o

    o.lib()
    work = []
    for j, (key, icb, pt, got) in enumerate(jobs):
        assert len(pt) == len(got)
        for off in range(0, max(len(pt), 1), window):
            work.append((j, off, min(window, len(pt) - off)))

    def one(wk):
        j, off, n = wk
        key, icb, pt, got = jobs[j]
        if n <= 0:
            return 0
        want = np.empty(n, dtype=np.uint8)
        src = np.ascontiguousarray(pt[off:off + n])
        o.ctr_into(key, icb, src.ctypes.data, want.ctypes.data, n, off // 16)
        return 0 if np.array_equal(want, got[off:off + n]) else 1

    cores = max(1, len(os.sched_getaffinity(0)))
    with cf.ThreadPoolExecutor(cores) as ex:
        bad = sum(ex.map(one, work))
    return sum(len(j[2]) for j in jobs), bad


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w, keybits = make_workload(args.workload)
    cores = len(os.sched_getaffinity(0))
    # requests per step: the whole workload when steps + warm-up of it fit a few minutes, else a bounded prefix
    per_step = oracle_requests_per_pass(w, keybits, cores, args.steps + args.warmup)
    src = oracle_sample(w, per_step)
    for _ in range(args.warmup):
        oracle_throughput(w, keybits, per_step, cores, src)
    t_total, b_total, per = 0.0, 0, []
    for _ in range(args.steps):
        gbs, dt = oracle_throughput(w, keybits, per_step, cores, src)
        t_total += dt
        per.append(dt)
        b_total += per_step * int(w.length[0])
    value = b_total / t_total / 1e9
    sample = "%d of the %d requests of %s per step (%d MiB), %d threads" % (
        per_step, w.n, w.name, per_step * int(w.length[0]) // MIB, cores)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps,
        "ms_per_step_median": 1e3 * float(np.median(per)), "ms_per_step_min": 1e3 * min(per), "ms_per_step_max": 1e3 * max(per),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": w.name, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))
    return 0


# --------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--backend", default="engine", choices=["engine", "launch"])
    ap.add_argument("--workload", default="c2", choices=["c2", "c3"])
    ap.add_argument("--chunk-rows", type=int, default=0)
    ap.add_argument("--mode", default="ctr", choices=["ctr", "ecb_encrypt", "ecb_decrypt", "cbc_decrypt"],
                    help="--backend launch only: what every request of the batch computes (SURVEY.md section 8(f3)); the vehicle of "
                         "the ncu captures of the other modes.  Their parity is tests/test_gpu_modes.py's; the oracle check of the "
                         "timed output is CTR's and is skipped for them")
    ap.add_argument("--launch-requests", type=int, default=0,
                    help="--backend launch: requests per ordinary launch (0 = the config's in-flight window; the whole "
                         "batch in ONE launch is the operating point the ncu captures under profiles/ are made at)")
    ap.add_argument("--no-extras", action="store_true", help="skip e2e / latency / cpu_baseline / kernel-only legs")
    ap.add_argument("--no-verify", action="store_true", help="skip the oracle check of the timed region's output (profiling runs)")
    ap.add_argument("--table2", action="store_true",
                    help="the paper's Table 2 (PAPER.md:356-369): 4 KiB .. 8 MiB, blocking server against a 32-thread executor")
    ap.add_argument("--sweep", action="store_true", help="configs[4]: size x in-flight x key-size table (one GPU)")
    ap.add_argument("--sweep-sizes", default="", help="with --sweep: comma-separated log2 sizes instead of 10..26")
    ap.add_argument("--sweep-out", default="", help="with --sweep / --openloop: also write the table to this JSON file")
    ap.add_argument("--openloop", action="store_true", help="latency under Poisson load, blocking vs overlapping (PAPER.md:244)")
    ap.add_argument("--openloop-bytes", type=int, default=4096)
    ap.add_argument("--dispatchers", type=int, default=0, help="with --dispatch-stats: dispatcher warps of the engine (0 = the default)")
    ap.add_argument("--dispatch-stats", action="store_true",
                    help="tuning aid, needs a library built with AESOFF_NVCC_EXTRA=-DAESOFF_DISP_STATS: what the dispatcher warps did "
                         "(requests per take, time from a poll landing to the token, time from the token to the last ticket) "
                         "while fine-grained cells ran under load")
    ap.add_argument("--plumbing-check", action="store_true",
                    help="run only the N-rank bookkeeping (rank discovery, host barrier, max-over-ranks reduction) on gloo, "
                         "no GPU work: what the CPU tests drive with two ranks")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    if args.openloop:
        return run_openloop(args)
    if args.table2:
        return run_table2(args)
    if args.dispatch_stats:
        return run_dispatch_stats(args)
    if args.warmup < 3:
        args.warmup = 3
    if args.mode != "ctr":
        if args.backend != "launch":
            raise SystemExit("bench.py: --mode needs --backend launch")
        args.no_verify = args.no_extras = True
    if args.plumbing_check:
        return plumbing_check(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)

    import torch
    import torch.distributed as dist

    import paper_2607_02630_b200.binding as B
    from paper_2607_02630_b200 import multi

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but %d rank(s) were launched: n_gpus would lie" % (args.gpus, world))
    if torch.cuda.device_count() <= local_rank:
        raise SystemExit("bench.py: rank %d has no GPU of its own (%d visible)" % (rank, torch.cuda.device_count()))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    host_pg = multi.host_group(dist) if world > 1 else None

    def barrier():
        if world > 1:
            dist.barrier()

    def barrier_host():
        # while the persistent kernel runs, a NCCL barrier kernel may find no free SM resources on a
        # full GPU: ranks line up through the store-based (host-side) barrier instead
        multi.host_barrier(dist, host_pg)

    hbm_peak, sm_max_mhz, peak_kind = _peaks()
    w, keybits = make_workload(args.workload)
    size = int(w.length[0])
    n = w.n

    # ---- device-resident payloads (2 x n x size bytes: far larger than the 126 MB L2) ----
    src = torch.empty(n * size, dtype=torch.uint8, device=dev)
    dst = torch.empty(n * size, dtype=torch.uint8, device=dev)
    stage = torch.empty(size, dtype=torch.uint8).pin_memory()
    for i in range(n):
        stage.numpy()[:] = w.payload(i)  # every rank uses the same seeded batch (weak scaling)
        src[i * size:(i + 1) * size].copy_(stage)
        torch.cuda.current_stream().synchronize()
    dst.zero_()
    torch.cuda.synchronize()
    # marshalled once (uint64 arrays go through the binding without a copy): the timed steps do no
    # per-request Python work
    srcs = np.asarray([src.data_ptr() + i * size for i in range(n)], dtype=np.uint64)
    dsts = np.asarray([dst.data_ptr() + i * size for i in range(n)], dtype=np.uint64)
    lens = np.asarray([size] * n, dtype=np.uint64)
    ctx = B.aes_ctx_create(w.key_of(0))
    side = torch.cuda.Stream(device=dev)
    launches0 = B.aes_engine_info()["kernel_launches"]

    # marshalled ONCE: a timed step is one call into the library (the closed loop over the batch), nothing else
    run_batch = B.aes_loop_prepare(w.icb, srcs, dsts, lens, window=w.in_flight, ctx=ctx)

    step_ms = []  # duration of each timed step: the library's own clock around the batch (engine), CUDA events (launch)

    def step_engine(timed=False):
        el, _, done = run_batch()
        assert done == n
        if timed:
            step_ms.append(el * 1e-6)

    LB = args.launch_requests or w.in_flight  # requests per ordinary launch in the launch backend

    def step_launch(stream_ptr, events=None):
        for b0 in range(0, n, LB):
            b1 = min(n, b0 + LB)
            if events is not None:
                e0 = torch.cuda.Event(enable_timing=True)
                e0.record()
            if args.mode == "ctr":
                B.aes_ctr_launch_batch([ctx] * (b1 - b0), w.icb[b0:b1], srcs[b0:b1], dsts[b0:b1], lens[b0:b1],
                                       device=local_rank, cuda_stream=stream_ptr, chunk_rows=args.chunk_rows)
            else:
                mode = {"ecb_encrypt": B.AES_MODE_ECB_ENC, "ecb_decrypt": B.AES_MODE_ECB_DEC, "cbc_decrypt": B.AES_MODE_CBC_DEC}[args.mode]
                B.aes_mode_launch_batch([mode] * (b1 - b0), [ctx] * (b1 - b0), w.icb[b0:b1], srcs[b0:b1], dsts[b0:b1], lens[b0:b1],
                                        device=local_rank, cuda_stream=stream_ptr, chunk_rows=args.chunk_rows)
            if events is not None:
                e1 = torch.cuda.Event(enable_timing=True)
                e1.record()
                events.append((e0, e1, (b1 - b0) * size))

    # ---- warm-up ----
    if args.backend == "engine":
        B.aes_engine_start(local_rank, chunk_rows=args.chunk_rows, idle_exit_ms=30000)
        for _ in range(args.warmup):
            step_engine()
        B.aes_engine_stop()
    else:
        for _ in range(args.warmup):
            step_launch(torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    barrier()

    # ---- timed region: exactly K steps ----
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kernel_events = []
    launches_before = B.aes_engine_info()["kernel_launches"]
    engine_start_ms = None
    with ClockSampler(local_rank) as clocks:
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        if args.backend == "engine":
            # step a0 (engine start: one launch, table fill) happens once per process, not per batch:
            # it sits outside the timed region like any other set-up, and is reported beside it
            ts0 = time.perf_counter()
            B.aes_engine_start(local_rank, chunk_rows=args.chunk_rows, idle_exit_ms=30000)
            engine_start_ms = 1e3 * (time.perf_counter() - ts0)
            barrier_host()
            t0 = time.perf_counter()
            ev0.record(side)
            for _ in range(args.steps):
                step_engine(timed=True)
            ev1.record(side)
            side.synchronize()
            t1h = time.perf_counter()
            B.aes_engine_stop()
        else:
            ev0.record()
            step_marks = [ev0]
            for _ in range(args.steps):
                step_launch(torch.cuda.current_stream().cuda_stream, kernel_events)
                step_marks.append(torch.cuda.Event(enable_timing=True))
                step_marks[-1].record()
            ev1.record()
        torch.cuda.synchronize()
        t1 = time.perf_counter() if args.backend != "engine" else t1h
    barrier()
    worker_stats = None
    if args.backend == "engine":
        # -DAESOFF_WSTATS builds only (AESOFF_NVCC_EXTRA=-DAESOFF_WSTATS python -m paper_2607_02630_b200.build --force): what the
        # worker warps of the persistent engine did during the K timed steps, from their own clock64 counters
        import ctypes

        ws = (ctypes.c_uint64 * 3)()
        if B._lib.aesoff_debug_worker_stats(local_rank, ws) == 0 and ws[2]:
            worker_stats = {"in_units_frac": ws[0] / float(ws[0] + ws[1]), "waiting_between_units_frac": ws[1] / float(ws[0] + ws[1]),
                            "units": int(ws[2]), "clocks_per_unit": ws[0] / float(ws[2]),
                            "how": "clock64 per worker warp: inside units / between two units, first unit to last unit of the engine run"}
    gpu_launches = B.aes_engine_info()["kernel_launches"] - launches_before
    ms_dev = ev0.elapsed_time(ev1)
    ms_host = 1e3 * (t1 - t0)
    if args.backend != "engine":
        step_ms = [a.elapsed_time(b) for a, b in zip(step_marks[:-1], step_marks[1:])]
    # replicas only: every rank ran the same batch on its own engine; the job
    # took as long as its slowest rank
    bps, ms_total = multi.job_throughput(ms_dev, n * size * args.steps, dist if world > 1 else None, host_pg)
    value = bps / 1e9
    clk = clocks.summary()

    # ---- parity of what the timed region wrote: EVERY byte of the last step's output against the oracle (rank 0;
    #      the oracle is test infrastructure and runs after the timed region, on the host cores) ----
    verified, verified_bytes = None, 0
    if rank == 0 and not args.no_verify:
        out_h = dst.cpu().numpy()
        jobs = [(w.key_of(i), w.icb_of(i), w.payload(i), out_h[i * size:(i + 1) * size]) for i in range(n)]
        verified_bytes, bad = verify_against_oracle(jobs)
        verified = bad == 0
        del out_h, jobs

    # ---- roofline of the dominant kernel (aesoff_engine_kernel) ----
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_mhz = clk["sm_mhz"] or sm_max_mhz
    lds_peak = SMEM_BYTES_PER_CLK_PER_SM * sm_count * sm_mhz * 1e6 / 1e9      # GB/s of lookup bytes
    lds_per_payload_byte = LOOKUPS[keybits] * 4.0 / 16.0
    if args.backend == "engine":
        kern_payload_gbs = n * size * args.steps / (ms_dev * 1e-3) / 1e9
        how = ("persistent kernel: one launch (aes_engine_start, outside the timed region) serves all K steps; achieved = "
               "algorithmic lookup bytes of the K steps / CUDA-event time of the K steps (events on a side stream)")
        kernel_ms = ms_dev
    else:
        per = [(e0.elapsed_time(e1), nb) for e0, e1, nb in kernel_events]
        kernel_ms = float(np.mean([p[0] for p in per]))
        kern_payload_gbs = float(np.mean([p[1] for p in per])) / (kernel_ms * 1e-3) / 1e9
        how = "ordinary launches of %d requests; mean CUDA-event time per launch on the launching stream" % LB
    roofline = {
        "bound": "alu", "unit_detail": "shared-memory lookup crossbar (LSU), 4-byte lookups",
        "kernel": "aesoff_engine_kernel",
        "achieved": kern_payload_gbs * lds_per_payload_byte, "peak": lds_peak, "unit": "GB/s",
        "frac": kern_payload_gbs * lds_per_payload_byte / lds_peak,
        "peak_how": "128 B/clk/SM x %d SMs x %.0f MHz (SM clock sampled in the run)" % (sm_count, sm_mhz),
        "lookups_per_block": LOOKUPS[keybits], "payload_gbs": kern_payload_gbs,
        "hbm": {"achieved": 2 * kern_payload_gbs, "peak": hbm_peak, "unit": "GB/s",
                "frac": 2 * kern_payload_gbs / hbm_peak, "peak_kind": peak_kind},
        "traffic": _ncu_traffic(args.workload)[0], "traffic_how": _ncu_traffic(args.workload)[1],
        ("timed_region_ms" if args.backend == "engine" else "avg_launch_ms"): kernel_ms, "how": how,
    }

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        # this rank's K steps one by one ("report the median run"); value and ms_per_step above are
        # the contract's: all K steps in one bracket, max over ranks
        "ms_per_step_median": float(np.median(step_ms)), "ms_per_step_min": float(min(step_ms)), "ms_per_step_max": float(max(step_ms)),
        "value_at_median_step": n * size / (float(np.median(step_ms)) * 1e-3) / 1e9,
        "dtype": "u8", "data": "synthetic",
        "config": {"workload": w.name if args.mode == "ctr" else w.name + "_" + args.mode, "backend": args.backend, "keybits": keybits, "request_bytes": size,
                   "requests_per_step": n, "in_flight": w.in_flight, "payload": "device-resident (HBM)",
                   "l2": "inputs larger than L2 (%.1f GiB src + same dst per step)" % (n * size / 2**30),
                   "seed": workloads.SEED_BASE + w.config_index},
        "gpu_launches": int(gpu_launches), "ms_host": ms_host, "engine_start_ms": engine_start_ms,
        "verified_vs_oracle": verified, "verified_bytes": verified_bytes, "worker_stats": worker_stats,
        "clocks": clk, "roofline": roofline,
    }

    if not args.no_extras and rank == 0 and world == 1:
        out.update(extras(args, B, torch, dev, local_rank, w, keybits, ctx, srcs, dsts, lens, size, n, step_launch,
                          lds_per_payload_byte, lds_peak, hbm_peak))
    elif not args.no_extras and world > 1:
        # every rank its own pinned buffers and engine; the oracle once, on rank 0 (so that a scaling record has both)
        e2e, held = e2e_leg(args, B, torch, dev, local_rank, w, ctx, lens, size, n, dist, host_pg)
        B.aes_engine_stop()
        for hp in held:
            B.aes_host_free(hp)
        if rank == 0:
            out["e2e"] = e2e
            out.update(cpu_baseline_leg(w, keybits, size, n))
    elif rank == 0:
        out["e2e"] = None
    if rank == 0:
        print(json.dumps(out))
    B.aes_ctx_destroy(ctx)
    if world > 1:
        dist.destroy_process_group()
    return 0


def plumbing_check(args):
    """The rank logic of our arm without its GPU work: every rank must find world == --gpus (a line that says
    n_gpus: N must come from N ranks), ranks line up through the host-side (gloo) barrier that is used while the
    persistent engines own the SMs, per-rank times reduce to the maximum and bytes to the sum; rank 0 prints."""
    import torch.distributed as dist

    from paper_2607_02630_b200 import multi

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but %d rank(s) were launched: n_gpus would lie" % (args.gpus, world))
    if world > 1:
        dist.init_process_group("gloo")
    g = multi.host_group(dist) if world > 1 else None
    multi.host_barrier(dist, g)
    bps, ms = multi.job_throughput(10.0 + rank, 10**9, dist if world > 1 else None, g)
    multi.host_barrier(dist, g)
    if rank == 0:
        print(json.dumps({"plumbing_check": True, "n_gpus": world, "ms_max": ms, "value": bps / 1e9, "unit": UNIT,
                          "scaling": "weak", "local_rank": int(os.environ.get("LOCAL_RANK", "0"))}))
    if world > 1:
        dist.destroy_process_group()
    return 0


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: one rank per GPU through torch.distributed.run on this
    node (replicas only); rank 0's JSON line is the job's.  Refuses to run when the
    node has fewer than N GPUs -- a line that says n_gpus: N must have used N."""
    import socket
    import subprocess

    import torch

    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit("bench.py: --gpus %d but this node has %d GPU(s)" % (args.gpus, have))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def mix_c4(B, torch, dev, n=10000, threads=(1, 4)):
    """BASELINE.json configs[3] on the running engine: 10,000 requests, sizes log-uniform 1-64 KiB with
    0-15 B tails, a fresh AES-128 or AES-256 key per request (aes_ctx_create inside the timed loop; the raw
    key rides in the descriptor and is expanded by the dispatcher warp that takes the request), random ICBs,
    256 in flight; from one executor thread and from four (the paper's
    executor is a pool).  Each variant is the median of five runs with its spread; the figures at the top level are those of
    the variant with the higher median, each variant is listed."""
    w4 = workloads.config4(n=n)
    stride = 64 * 1024 + 16
    s4 = torch.empty(n * stride, dtype=torch.uint8, device=dev)  # contents are irrelevant to timing
    d4 = torch.empty(n * stride, dtype=torch.uint8, device=dev)
    keys = np.zeros((n, 32), dtype=np.uint8)
    kb = np.zeros(n, dtype=np.int32)
    for i in range(n):
        k = w4.key_of(i)
        keys[i, :len(k)] = np.frombuffer(k, dtype=np.uint8)
        kb[i] = 8 * len(k)
    srcs = np.asarray([s4.data_ptr() + i * stride for i in range(n)], dtype=np.uint64)
    dsts = np.asarray([d4.data_ptr() + i * stride for i in range(n)], dtype=np.uint64)
    out = {"workload": w4.name, "requests": n, "in_flight": w4.in_flight, "mean_bytes": float(w4.length.mean()),
           "key_expansion": "per request, on the device", "variants": {}}
    for th in threads:
        B.aes_loop_run(w4.icb, srcs, dsts, w4.length, window=w4.in_flight, keys=keys, keybits=kb, want_latency=False, threads=th)
        runs = []
        for _ in range(5):
            r = B.aes_loop_run(w4.icb, srcs, dsts, w4.length, window=w4.in_flight, keys=keys, keybits=kb, threads=th)
            a = r["lat_ns"][n // 20:] / 1e3
            runs.append({"p50_us": percentile(a, 50), "p99_us": percentile(a, 99), "req_per_s": n / (r["elapsed_ns"] * 1e-9),
                         "payload_gbs": r["bytes"] / r["elapsed_ns"]})
        out["variants"]["executor_threads_%d" % th] = median_run(runs, "req_per_s")
    top = max(out["variants"].values(), key=lambda v: v["req_per_s"])
    out.update(top)
    return out


def extra_cells(B, torch, dev, lds_peak, hbm_peak):
    """Sweep cells that belong in the driver-run record: the metric's "8 MiB" half -- BASELINE.json configs[2]
    (AES-256, 200 x 8 MiB, 16 in flight, every byte of 16 requests and the first and last 64 KiB of the others checked)
    and the AES-128 8 MiB cell -- lone large requests (the paper's single-op column, Table 2 at PAPER.md:356-369), and
    the fine-grained cells from one and from four executor threads."""
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE + 8, 1]))
    out = {}
    # configs[2] out of place, seeded payloads, verified
    w3 = workloads.config3()
    size, n = int(w3.length[0]), w3.n
    src = torch.empty(n * size, dtype=torch.uint8, device=dev)
    dst = torch.empty(n * size, dtype=torch.uint8, device=dev)
    stage = torch.empty(size, dtype=torch.uint8).pin_memory()
    for i in range(n):
        stage.numpy()[:] = w3.payload(i)
        src[i * size:(i + 1) * size].copy_(stage)
        torch.cuda.current_stream().synchronize()
    srcs = np.asarray([src.data_ptr() + i * size for i in range(n)], dtype=np.uint64)
    dsts = np.asarray([dst.data_ptr() + i * size for i in range(n)], dtype=np.uint64)
    ctx3 = B.aes_ctx_create(w3.key_of(0))
    B.aes_loop_run(w3.icb, srcs, dsts, w3.length, window=w3.in_flight, ctx=ctx3, want_latency=False)
    c3runs = []
    for _ in range(5):
        r = B.aes_loop_run(w3.icb, srcs, dsts, w3.length, window=w3.in_flight, ctx=ctx3, want_latency=False)
        c3runs.append({"payload_gbs": r["bytes"] / r["elapsed_ns"]})
    c3med = median_run(c3runs, "payload_gbs")
    best = c3med["payload_gbs"]
    out_h = dst.cpu().numpy()
    jobs, W = [], 64 * 1024
    for i in range(n):
        pt, got = w3.payload(i), out_h[i * size:(i + 1) * size]
        if i % 13 == 0:
            jobs.append((w3.key_of(i), w3.icb_of(i), pt, got))
        else:
            from oracle import oracle as o  # test infrastructure, after the timed runs
            for off in (0, size - W):
                jobs.append((w3.key_of(i), o.ctr_add(w3.icb_of(i), off // 16), pt[off:off + W], got[off:off + W]))
    vb, bad = verify_against_oracle(jobs)
    out["c3_aes256_8MiB_x200_w16"] = {"workload": w3.name, "payload_gbs": best, "runs": 5, "payload_gbs_min": c3med["payload_gbs_min"],
                                      "payload_gbs_max": c3med["payload_gbs_max"],
                                      "frac_lookup_roof": best * LOOKUPS[256] / 4.0 / lds_peak, "frac_hbm_roof": 2 * best / hbm_peak,
                                      "verified_bytes": vb, "verified_vs_oracle": bad == 0}
    B.aes_ctx_destroy(ctx3)
    del out_h, jobs
    # in-place cells over the same memory (timing only; the per-cell parity batches are bench.py --sweep's)
    base, pool_bytes = src.data_ptr(), n * size
    ctx = B.aes_ctx_create(rng.bytes(16))

    def cell(size, depth, nreq, threads=1, reps=3):
        nbuf = max(1, min(pool_bytes // size, max(depth, 64)))
        ptrs = np.asarray([base + (i % nbuf) * size for i in range(nreq)], dtype=np.uint64)
        icb = rng.integers(0, 256, size=(nreq, 16), dtype=np.uint8)
        lens = np.full(nreq, size, dtype=np.uint64)
        B.aes_loop_run(icb[:2 * depth], ptrs[:2 * depth], ptrs[:2 * depth], lens[:2 * depth], window=depth, ctx=ctx, want_latency=False)
        c = run_cell(B, ptrs, icb, lens, depth, ctx, threads=threads, reps=reps)
        c["frac_lookup_roof"] = c["payload_gbs"] * LOOKUPS[128] / 4.0 / lds_peak
        c["frac_hbm_roof"] = 2 * c["payload_gbs"] / hbm_peak
        return c

    out["aes128_8MiB_w16"] = cell(8 * MIB, 16, 1000)
    out["aes128_1MiB_w16"] = cell(MIB, 16, 8000)
    for sz, name in ((MIB, "1MiB"), (4 * MIB, "4MiB"), (8 * MIB, "8MiB"), (64 * MIB, "64MiB")):
        out["aes128_%s_w1" % name] = cell(sz, 1, 1000 if sz <= 8 * MIB else 150)
    for sz, name in ((4096, "4KiB"), (65536, "64KiB")):
        for th in (1, 4):
            out["aes128_%s_w256_threads%d" % (name, th)] = cell(sz, 256, 150000, threads=th)
            out["aes128_%s_w1024_threads%d" % (name, th)] = cell(sz, 1024, 150000, threads=th)
    # the other modes at the headline shape: 1 MiB requests, 64 in flight, out of place
    nreq = 4000
    nbuf = 128
    icb = rng.integers(0, 256, size=(nreq, 16), dtype=np.uint8)
    lens = np.full(nreq, MIB, dtype=np.uint64)
    ps = np.asarray([base + (i % nbuf) * MIB for i in range(nreq)], dtype=np.uint64)
    pd = np.asarray([base + (nbuf + i % nbuf) * MIB for i in range(nreq)], dtype=np.uint64)
    for name, mode in (("ecb_encrypt", B.AES_MODE_ECB_ENC), ("ecb_decrypt", B.AES_MODE_ECB_DEC), ("cbc_decrypt", B.AES_MODE_CBC_DEC)):
        B.aes_loop_run(icb[:128], ps[:128], pd[:128], lens[:128], window=64, ctx=ctx, want_latency=False, mode=mode)
        r = B.aes_loop_run(icb, ps, pd, lens, window=64, ctx=ctx, want_latency=False, mode=mode)
        out["aes128_%s_1MiB_w64" % name] = {"payload_gbs": r["bytes"] / r["elapsed_ns"], "frac_hbm_roof": 2 * r["bytes"] / r["elapsed_ns"] / hbm_peak}
    B.aes_ctx_destroy(ctx)
    return out


def median_run(runs, key):
    """The median run of a repeated cell by `key` (the upper one of an even count), with the spread beside it: a best-of
    figure is biased upward and hides the spread."""
    order = sorted(runs, key=lambda v: v[key])
    v = dict(order[len(order) // 2])
    v["runs"] = len(runs)
    v[key + "_min"], v[key + "_max"] = order[0][key], order[-1][key]
    return v


def run_cell(B, ptrs, icb, lens, depth, ctx, threads=1, reps=1):
    """One closed-loop run of equal-sized requests on the running engine -> dict (the median of `reps` runs by throughput)."""
    n = len(lens)
    runs = []
    for _ in range(reps):
        r = B.aes_loop_run(icb, ptrs, ptrs, lens, window=depth, ctx=ctx, threads=threads)
        a = r["lat_ns"][n // 20:] / 1e3
        runs.append({"payload_gbs": r["bytes"] / r["elapsed_ns"], "req_per_s": n / (r["elapsed_ns"] * 1e-9),
                     "p50_us": percentile(a, 50), "p99_us": percentile(a, 99)})
    return median_run(runs, "payload_gbs")


def verify_cell(B, torch, dev, size, depth, keybits, key, ctx, rng, budget=64 * MIB):
    """SURVEY.md section 8(d) parity coverage of a sweep cell: min(depth, budget / size) >= 1 requests of this size,
    all in flight together, out of place from a seeded payload, every byte against the oracle.  -> (bytes, ok)."""
    m = int(max(1, min(depth, budget // size)))
    host = rng.integers(0, 256, size=m * size, dtype=np.uint8)
    src = torch.empty(m * size, dtype=torch.uint8, device=dev)   # allocations come from torch's cache: no cudaMalloc
    dst = torch.empty(m * size, dtype=torch.uint8, device=dev)   # (which would wait for the persistent kernel)
    src.copy_(torch.from_numpy(host))
    torch.cuda.current_stream().synchronize()
    icb = rng.integers(0, 256, size=(m, 16), dtype=np.uint8)
    srcs = np.asarray([src.data_ptr() + i * size for i in range(m)], dtype=np.uint64)
    dsts = np.asarray([dst.data_ptr() + i * size for i in range(m)], dtype=np.uint64)
    r = B.aes_loop_run(icb, srcs, dsts, np.full(m, size, dtype=np.uint64), window=depth, ctx=ctx, want_latency=False)
    assert r["requests"] == m
    out = dst.cpu().numpy()
    jobs = [(key, icb[i].tobytes(), host[i * size:(i + 1) * size], out[i * size:(i + 1) * size]) for i in range(m)]
    nbytes, bad = verify_against_oracle(jobs)
    return nbytes, bad == 0


def run_sweep(args):
    """BASELINE.json configs[4]: payload 1 KiB .. 64 MiB in powers of two x in-flight 1/16/256/1024, AES-128 and
    AES-256, on the persistent engine; one JSON object per cell to stdout (and --sweep-out).  Timing runs in place
    over an 8 GiB pool (a cell whose depth x size exceeds it reuses buffers among the requests in flight and says
    so); parity is checked per cell by a separate out-of-place batch of the same shape (verify_cell)."""
    import torch

    import paper_2607_02630_b200.binding as B

    hbm_peak, sm_max_mhz, _ = _peaks()
    dev = torch.device("cuda", 0)
    total = 8 << 30
    buf = torch.empty(total, dtype=torch.uint8, device=dev)
    buf.random_(0, 256)
    warm = torch.empty(2 * 64 * MIB, dtype=torch.uint8, device=dev)  # puts the verification buffers into torch's cache
    del warm
    torch.cuda.synchronize()
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    lds_peak = SMEM_BYTES_PER_CLK_PER_SM * sm_count * sm_max_mhz * 1e6 / 1e9
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE + 5, 1]))
    cells = []
    sizes = range(10, 27) if not args.sweep_sizes else [int(x) for x in args.sweep_sizes.split(",")]
    B.aes_engine_start(0, idle_exit_ms=60000)
    try:
        for keybits in (128, 256):
            key = rng.bytes(keybits // 8)
            ctx = B.aes_ctx_create(key)
            for lg in sizes:
                size = 1 << lg
                for depth in (1, 16, 256, 1024):
                    nbuf = max(1, min(total // size, max(depth, 64)))
                    shared = nbuf < depth  # 64 MiB x 256 / 1024: more in flight than distinct buffers fit
                    # about 50 ms of work per cell, from a rough rate estimate
                    rate = min(600e9 / size, 8e6, depth / 10e-6)
                    n = int(min(max(0.05 * rate, 4 * depth, 64), 400000))
                    ptrs = np.asarray([buf.data_ptr() + (i % nbuf) * size for i in range(n)], dtype=np.uint64)
                    icb = np.zeros((n, 16), dtype=np.uint8)
                    icb[:, :8] = rng.integers(0, 256, size=(n, 8), dtype=np.uint8)
                    lens = np.full(n, size, dtype=np.uint64)
                    w = min(n, depth * 2)
                    B.aes_loop_run(icb[:w], ptrs[:w], ptrs[:w], lens[:w], window=depth, ctx=ctx, want_latency=False)
                    cell = {"keybits": keybits, "bytes": size, "in_flight": depth, "requests": n, "in_place": True,
                            "buffers_shared_among_in_flight": shared}
                    cell.update(run_cell(B, ptrs, icb, lens, depth, ctx))
                    if depth >= 256 and size <= 256 * 1024:
                        # the fine-grained regime from a pool of executor threads as well
                        cell["executor_threads_4"] = run_cell(B, ptrs, icb, lens, depth, ctx, threads=4)
                    gbs = cell["payload_gbs"]
                    cell["frac_lookup_roof"] = gbs * LOOKUPS[keybits] * 4.0 / 16.0 / lds_peak
                    cell["frac_hbm_roof"] = 2 * gbs / hbm_peak
                    vb, ok = verify_cell(B, torch, dev, size, depth, keybits, key, ctx, rng)
                    cell["verified_bytes"], cell["verified_vs_oracle"] = vb, ok
                    cells.append(cell)
                    print(json.dumps(cell), flush=True)
            B.aes_ctx_destroy(ctx)
    finally:
        B.aes_engine_stop()
    if args.sweep_out:
        with open(args.sweep_out, "w") as f:
            json.dump({"lookup_roof_gbs_of_lookup_bytes": lds_peak, "hbm_peak_gbs": hbm_peak, "sm_mhz_assumed": sm_max_mhz,
                       "note": "timing in place over an 8 GiB pool; parity per cell: min(depth, 64 MiB / size) >= 1 requests "
                               "of the cell's shape out of place, every byte against the oracle (verified_bytes)",
                       "cells": cells}, f, indent=1)
    return 0 if all(c["verified_vs_oracle"] for c in cells) else 1


def run_table2(args):
    """The paper's Appendix A sweep (Table 2; Fig. 11 at PAPER.md:240) with the real engine:
    block sizes 4 KiB .. 8 MiB, AES-128-CTR, 50 logical clients.  'sync' is the server the paper starts from: it
    waits for each offload, so one request is in flight (aes_loop_run, window 1).  'async' is the rerouted server:
    a 32-thread executor, each thread blocking on its own offload, so up to 32 are in flight
    (aes_loop_run_mt, 32 threads, window 32).  Payloads device-resident and, as in the paper (j.buf is host memory,
    PAPER.md:132), in pinned host memory.  Context beside the paper's numbers (another GPU, another server), not a target."""
    import torch

    import paper_2607_02630_b200.binding as B

    paper = {4096: (46.4, 3750, 4667), 8192: (47.0, None, None), 16384: (51.4, None, None), 32768: (60.3, None, None),
             65536: (70.2, None, None), 131072: (92.7, None, None), 262144: (126.5, None, None), 524288: (191.8, None, None),
             1 << 20: (361.6, 1538, 3644), 2 << 20: (653.6, None, None), 4 << 20: (1188.1, None, None), 8 << 20: (2258.6, 227, 1228)}
    dev = torch.device("cuda", 0)
    pool = 64
    buf = torch.empty(pool * (8 << 20), dtype=torch.uint8, device=dev)
    buf.random_(0, 256)
    torch.cuda.synchronize()
    hbuf = B.aes_host_alloc(pool * (8 << 20))
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE + 7, 1]))
    ctx = B.aes_ctx_create(rng.bytes(16))
    rows = []
    B.aes_engine_start(0, idle_exit_ms=60000)
    try:
        for lg in range(12, 24):
            size = 1 << lg
            row = {"bytes": size, "paper_us": paper[size][0], "paper_sync_req_s": paper[size][1], "paper_async_req_s": paper[size][2]}
            for where, base in (("device", buf.data_ptr()), ("host", hbuf)):
                n1 = int(min(4000, max(200, 0.05 / (10e-6 + size / 400e9))))
                ptrs = np.asarray([base + (i % pool) * size for i in range(n1 * 8)], dtype=np.uint64)
                icb = rng.integers(0, 256, size=(n1 * 8, 16), dtype=np.uint8)
                lens = np.full(n1 * 8, size, dtype=np.uint64)
                B.aes_loop_run(icb[:64], ptrs[:64], ptrs[:64], lens[:64], window=1, ctx=ctx, want_latency=False)
                sync = run_cell(B, ptrs[:n1], icb[:n1], lens[:n1], 1, ctx)
                asyn = B.aes_loop_run(icb, ptrs, ptrs, lens, window=32, ctx=ctx, threads=32, want_latency=False)
                a_rps = len(lens) / (asyn["elapsed_ns"] * 1e-9)
                row[where] = {"single_op_us": sync["p50_us"], "sync_req_s": sync["req_per_s"], "async_req_s": a_rps,
                              "speedup": a_rps / sync["req_per_s"], "async_payload_gbs": asyn["bytes"] / asyn["elapsed_ns"]}
            rows.append(row)
            print(json.dumps(row), flush=True)
    finally:
        B.aes_engine_stop()
        B.aes_ctx_destroy(ctx)
        B.aes_host_free(hbuf)
    if args.sweep_out:
        with open(args.sweep_out, "w") as f:
            json.dump({"rows": rows}, f, indent=1)
    return 0


def run_dispatch_stats(args):
    """Where the dispatch pipeline's time goes under load (a request at 256 in flight takes twice as long as a
    lone one).  Per cell, on a fresh engine of a -DAESOFF_DISP_STATS build: the closed loop's rate and latency, and per
    dispatcher warp its polls that took requests ("takes"), requests per take, the time from a poll landing to the token
    arriving (parse, geometry and waiting for the dispatcher before it) and from the token to the last ticket store (key
    expansion, descriptor and ticket stores, fences), by the GPU's globaltimer."""
    import ctypes

    import torch

    import paper_2607_02630_b200.binding as B

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    torch.zeros(1, device=dev)
    torch.cuda.synchronize()
    get = B._lib.aesoff_debug_dispatch_stats
    get.restype, get.argtypes = ctypes.c_int, [ctypes.c_void_p]
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE + 9, 1]))
    pool = torch.empty(256 * MIB, dtype=torch.uint8, device=dev)
    ctx = B.aes_ctx_create(rng.bytes(16))

    def read_stats(ndisp):
        time.sleep(0.05)  # the counters reach the host-mapped words at the first empty poll after the run
        raw = (ctypes.c_uint32 * 40)()
        assert get(raw) == 0
        out = []
        for d in range(ndisp):
            takes, reqs, wait, work, empty = [int(raw[5 * d + i]) for i in range(5)]
            if takes == 0:
                continue
            out.append({"dispatcher": d, "takes": takes, "requests_per_take": reqs / takes, "wait_us_per_take": wait * 0.064 / takes,
                        "work_us_per_take": work * 0.064 / takes, "work_us_per_request": work * 0.064 / max(reqs, 1), "empty_polls": empty})
        return out

    cells = {}

    def fixed(name, size, depth, nreq, threads=1):
        B.aes_engine_start(0, idle_exit_ms=30000, n_dispatchers=args.dispatchers)
        nd = B.aes_engine_info()["n_dispatchers"]
        nbuf = max(depth, 64)
        ptrs = np.asarray([pool.data_ptr() + (i % nbuf) * size for i in range(nreq)], dtype=np.uint64)
        icb = rng.integers(0, 256, size=(nreq, 16), dtype=np.uint8)
        lens = np.full(nreq, size, dtype=np.uint64)
        c = run_cell(B, ptrs, icb, lens, depth, ctx, threads=threads, reps=3)
        c["in_flight"], c["executor_threads"] = depth, threads
        c["dispatchers"] = read_stats(nd)
        B.aes_engine_stop()
        cells[name] = c

    fixed("aes128_4KiB_w1", 4096, 1, 20000)
    fixed("aes128_4KiB_w256", 4096, 256, 150000)
    fixed("aes128_4KiB_w256_threads4", 4096, 256, 150000, threads=4)
    fixed("aes128_4KiB_w1024_threads4", 4096, 1024, 150000, threads=4)
    fixed("aes128_64KiB_w256", 65536, 256, 150000)
    for th in (1, 4):
        B.aes_engine_start(0, idle_exit_ms=30000, n_dispatchers=args.dispatchers)
        nd = B.aes_engine_info()["n_dispatchers"]
        m = mix_c4(B, torch, dev, threads=(th,))
        m["dispatchers"] = read_stats(nd)
        B.aes_engine_stop()
        cells["mix_c4_threads%d" % th] = m
    B.aes_ctx_destroy(ctx)
    if not any(c["dispatchers"] for c in cells.values()):
        raise SystemExit("bench.py --dispatch-stats: all counters are zero: build the library with "
                         "AESOFF_NVCC_EXTRA=-DAESOFF_DISP_STATS python -m paper_2607_02630_b200.build --force")
    out = {"dispatch_stats": cells, "how": run_dispatch_stats.__doc__.split("\n\n")[0].replace("\n    ", " ")}
    print(json.dumps(out))
    if args.sweep_out:
        with open(args.sweep_out, "w") as f:
            json.dump(out, f, indent=1)
    return 0


def run_openloop(args):
    """The paper's latency-under-load experiment (Fig. 12) with the REAL offload instead of the
    paper's 20 us emulated one: Poisson arrivals of 4 KiB AES-128-CTR requests at a swept offered load, one
    server thread that either waits for each offload (blocking) or keeps serving and polls (overlapping)."""
    import torch

    import paper_2607_02630_b200.binding as B

    dev = torch.device("cuda", 0)
    size, pool = args.openloop_bytes, 4096
    buf = torch.empty(2 * pool * size, dtype=torch.uint8, device=dev)
    buf.random_(0, 256)
    torch.cuda.synchronize()
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE + 6, 1]))
    ctx = B.aes_ctx_create(rng.bytes(16))
    rows = []
    B.aes_engine_start(0, idle_exit_ms=30000)
    try:
        for rate in (25e3, 50e3, 75e3, 100e3, 150e3, 200e3, 400e3, 800e3, 1.6e6, 2.4e6, 3.2e6, 4.0e6, 4.8e6):
            n = int(min(max(rate * 0.05, 2000), 200000))
            gaps = rng.exponential(1e9 / rate, size=n)
            arrival = np.cumsum(gaps).astype(np.uint64)
            icb = rng.integers(0, 256, size=(n, 16), dtype=np.uint8)
            srcs = np.asarray([buf.data_ptr() + (i % pool) * size for i in range(n)], dtype=np.uint64)
            dsts = np.asarray([buf.data_ptr() + (pool + i % pool) * size for i in range(n)], dtype=np.uint64)
            lens = np.full(n, size, dtype=np.uint64)
            row = {"offered_req_per_s": rate, "bytes": size, "requests": n}
            for mode in ("overlapping", "blocking"):
                r = B.aes_openloop_run(icb, srcs, dsts, lens, arrival, ctx, blocking=(mode == "blocking"))
                a = r["lat_ns"][n // 20:] / 1e3
                row[mode] = {"p50_us": percentile(a, 50), "p99_us": percentile(a, 99),
                             "achieved_req_per_s": n / (r["elapsed_ns"] * 1e-9), "max_in_flight": int(r["max_in_flight"]),
                             "ring_full": int(r["ring_full_spins"])}
            rows.append(row)
            print(json.dumps(row), flush=True)
    finally:
        B.aes_engine_stop()
        B.aes_ctx_destroy(ctx)
    if args.sweep_out:
        with open(args.sweep_out, "w") as f:
            json.dump({"rows": rows}, f, indent=1)
    return 0


def extras(args, B, torch, dev, local_rank, w, keybits, ctx, srcs, dsts, lens, size, n, step_launch,
           lds_per_payload_byte, lds_peak, hbm_peak):
    res = {}
    # ---- kernel-only leg: the worker code through ordinary launches, CUDA events per launch ----
    if args.backend == "engine":
        evs = []
        step_launch(torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        for _ in range(3):
            step_launch(torch.cuda.current_stream().cuda_stream, evs)
        torch.cuda.synchronize()
        ms = float(np.mean([a.elapsed_time(b) for a, b, _ in evs]))
        gbs = float(np.mean([nb for _, _, nb in evs])) / (ms * 1e-3) / 1e9
        res["kernel_only"] = {"backend": "launch", "requests_per_launch": w.in_flight, "avg_launch_ms": ms,
                              "payload_gbs": gbs, "lds_frac": gbs * lds_per_payload_byte / lds_peak,
                              "hbm_frac": 2 * gbs / hbm_peak, "launches_timed": len(evs)}

    # ---- the same batch as ONE closed loop over 10 passes: the window never drains between passes (a timed step above is
    #      the whole 1,000-request job, so it fills an idle GPU and drains it every time: DESIGN.md R14) ----
    if args.backend == "engine":
        B.aes_engine_start(local_rank, chunk_rows=args.chunk_rows, idle_exit_ms=30000)
        go = B.aes_loop_prepare(w.icb, srcs, dsts, lens, window=w.in_flight, ctx=ctx, repeat=10)
        go()
        el, by, _ = go()
        B.aes_engine_stop()
        res["steady_state"] = {"payload_gbs": by / el, "lds_frac": by / el * lds_per_payload_byte / lds_peak, "hbm_frac": 2 * by / el / hbm_peak,
                               "how": "the %d requests of the step, 10 passes back to back in one closed loop, %d in flight throughout" % (n, w.in_flight)}

    # ---- e2e: payloads in pinned HOST memory, read and written by the kernel over PCIe (leaves the engine running) ----
    e2e, (hs, hd) = e2e_leg(args, B, torch, dev, local_rank, w, ctx, lens, size, n)
    res["e2e"] = e2e

    # ---- latency at 4 KiB (the metric's second half), device-resident, 1 and 256 in flight ----
    lat = {}
    nl = 10000
    small = 4096
    pool = 512
    lsrc = torch.empty(pool * small, dtype=torch.uint8, device=dev)  # no kernel: contents are irrelevant to timing
    ldst = torch.empty(pool * small, dtype=torch.uint8, device=dev)
    wl = workloads.fixed_size(small, nl, 1)
    ls = [lsrc.data_ptr() + (i % pool) * small for i in range(nl)]
    ld = [ldst.data_ptr() + (i % pool) * small for i in range(nl)]
    for depth in (1, 256):
        r = B.aes_loop_run(wl.icb, ls, ld, [small] * nl, window=depth, ctx=ctx)
        a = r["lat_ns"][nl // 20:] / 1e3
        lat["inflight_%d" % depth] = {"p50_us": percentile(a, 50), "p99_us": percentile(a, 99),
                                      "mean_us": float(a.mean()), "req_per_s": nl / (r["elapsed_ns"] * 1e-9)}
    res["latency_4KiB"] = lat
    # ---- configs[0]: one 64 KiB AES-128 request, one in flight ----
    w1 = workloads.config1()
    n1 = 2000
    r = B.aes_loop_run(np.repeat(w1.icb, n1, axis=0), [lsrc.data_ptr()] * n1, [ldst.data_ptr()] * n1, [65536] * n1, window=1, ctx=ctx)
    a = r["lat_ns"][n1 // 20:] / 1e3
    res["c1_64KiB_single"] = {"workload": w1.name, "p50_us": percentile(a, 50), "p99_us": percentile(a, 99),
                              "payload_gbs": 65536.0 / (percentile(a, 50) * 1e3)}
    # same, payload in pinned HOST memory (the paper's j.buf): read and written over PCIe by the kernel
    hl = B.aes_host_alloc(2 * pool * small)
    hls = [hl + (i % pool) * small for i in range(nl)]
    hld = [hl + (pool + i % pool) * small for i in range(nl)]
    r = B.aes_loop_run(wl.icb, hls, hld, [small] * nl, window=1, ctx=ctx)
    a = r["lat_ns"][nl // 20:] / 1e3
    res["latency_4KiB"]["host_payload_inflight_1"] = {"p50_us": percentile(a, 50), "p99_us": percentile(a, 99),
                                                      "mean_us": float(a.mean())}
    # ---- the metric's 8 MiB half and the cells the round's targets are quoted on (all on the running engine) ----
    res["cells"] = extra_cells(B, torch, dev, lds_peak, hbm_peak)
    res["e2e"]["latency_4KiB"] = {k: {"p50_us": v["p50_us"], "p99_us": v["p99_us"]} for k, v in res["latency_4KiB"].items()}
    res["roofline_at_8MiB"] = {k: {f: c[f] for f in ("payload_gbs", "frac_lookup_roof", "frac_hbm_roof", "frac_alu_roof") if f in c}
                               for k, c in res["cells"].items() if k in ("aes128_8MiB_w16", "c3_aes256_8MiB_x200_w16")}
    # ---- configs[3]: the fine-grained mix, per-request keys (key expansion on the path) ----
    res["mix_c4"] = mix_c4(B, torch, dev)
    B.aes_engine_stop()
    B.aes_host_free(hl)
    # freeing pinned memory synchronises the device, so only after the engine has stopped
    B.aes_host_free(hs)
    B.aes_host_free(hd)

    # ---- calibration: what the lookup pipe, the ALU pipe and the payload path deliver on this GPU ----
    try:
        cal = B.aes_calibrate(local_rank)
        cal["lookup_pipe_frac_of_nominal"] = cal["lookups_per_clk_per_sm"] / 32.0
        cal["main_round_frac_of_nominal"] = cal["round_lookups_per_clk_per_sm"] / 32.0
        # the bitsliced alternative: one warp-wide S-box evaluation covers 32 lanes x 32 bytes; an AES-128
        # block needs 160 byte substitutions; MixColumns, AddRoundKey and the bit transposes come on top and are NOT counted
        cal["bitslice_subbytes_only_aes128_gbs"] = (cal["bitslice_sboxes_per_clk_per_sm"] * 1024.0 * cal["sm_count"] *
                                                    cal["sm_mhz"] * 1e6 / 160.0 * 16.0 / 1e9)
        cal["bitslice_how"] = ("tower-field circuit generated and checked by csrc/gen_bitslice_sbox.py, 117 LOP3 per S-box in the SASS, "
                               "verified on all 256 inputs on the GPU (bitslice_mismatches must be 0), 4 independent chains per thread; "
                               "the figure is the ceiling of SubBytes ALONE for a bitsliced AES-128")
        cal["how"] = ("aes_calibrate: microkernels with the engine's table layout and launch shape; nominal = 32 lookups and "
                      "2 warp-wide ALU instructions per clock per SM (guides/B300_MICROARCH.md)")
        res["calibration"] = cal
    except Exception as e:  # noqa: BLE001
        res["calibration"] = {"error": str(e)}

    res.update(cpu_baseline_leg(w, keybits, size, n))
    return res


def e2e_leg(args, B, torch, dev, local_rank, w, ctx, lens, size, n, dist=None, host_pg=None):
    """The metric end to end through the public call with HOST buffers: src and dst in pinned host memory (aes_host_alloc), read
    and written by the kernel over PCIe inside the timed region; every output byte checked against the oracle afterwards (rank 0).
    Starts the engine and leaves it running.  With several ranks each has its own buffers and engine; the figure is all ranks'
    bytes over the slowest rank's time.  Returns (the e2e object, (src, dst) host allocations to free after the engine stops)."""
    from paper_2607_02630_b200 import multi

    n_e2e = min(n, 256)
    hs = B.aes_host_alloc(n_e2e * size)
    hd = B.aes_host_alloc(n_e2e * size)
    hsv, hdv = B.host_view(hs, n_e2e * size), B.host_view(hd, n_e2e * size)
    for i in range(n_e2e):
        hsv[i * size:(i + 1) * size] = w.payload(i)
    hsrcs = [hs + i * size for i in range(n_e2e)]
    hdsts = [hd + i * size for i in range(n_e2e)]
    pcie = pcie_roof(torch, dev, hsv, hdv, 32 * MIB)   # before the engine starts
    hdv[:] = 0
    B.aes_engine_start(local_rank, chunk_rows=args.chunk_rows, idle_exit_ms=30000)
    B.aes_loop_run(w.icb[:n_e2e], hsrcs, hdsts, lens[:n_e2e], window=w.in_flight, ctx=ctx, want_latency=False)
    reps = 4
    multi.host_barrier(dist, host_pg)
    t0 = time.perf_counter()
    r = B.aes_loop_run(w.icb[:n_e2e], hsrcs, hdsts, lens[:n_e2e], window=w.in_flight, ctx=ctx, repeat=reps,
                       want_latency=False)
    t1 = time.perf_counter()
    bps, _ = multi.job_throughput(1e3 * (t1 - t0), r["bytes"], dist, host_pg)
    e2e_gbs = bps / 1e9
    ranks = dist.get_world_size() if dist is not None else 1
    e2e = {"value": e2e_gbs, "unit": UNIT, "h2d_bytes_per_step": n_e2e * size * ranks, "d2h_bytes_per_step": n_e2e * size * ranks,
           "how": "aes_ctr_submit with src/dst in pinned host memory (aes_host_alloc): the kernel reads the "
                  "payload and writes the result over PCIe inside the timed region; %d requests x %d B, %d in "
                  "flight, %d repeats%s" % (n_e2e, size, w.in_flight, reps,
                                            "" if ranks == 1 else "; per rank, %d ranks, all bytes / slowest rank" % ranks)}
    if int(os.environ.get("RANK", "0")) == 0:
        e2e_vb, e2e_bad = verify_against_oracle([(w.key_of(i), w.icb_of(i), w.payload(i), hdv[i * size:(i + 1) * size])
                                                 for i in range(n_e2e)])
        e2e["verified_vs_oracle"], e2e["verified_bytes"] = bool(e2e_bad == 0), e2e_vb
    if pcie:
        # host-resident payloads are measured against the link, not against HBM (per GPU)
        per_gpu = e2e_gbs / ranks
        e2e["roofline"] = {"bound": "pcie", "achieved": per_gpu, "peak": pcie["both_ways_gbs_each"], "unit": "GB/s each way per GPU",
                           "frac": per_gpu / pcie["both_ways_gbs_each"], "peak_how": pcie["how"],
                           "h2d_alone_gbs": pcie["h2d_alone_gbs"], "d2h_alone_gbs": pcie["d2h_alone_gbs"]}
    del hsv, hdv
    return e2e, (hs, hd)


def cpu_baseline_leg(w, keybits, size, n):
    """cpu_baseline (the oracle, as it stands, on the host cores; all of the workload where that fits about 25 s, and a
    one-core figure) and the AES-NI context lines."""
    res = {}
    # ---- cpu_baseline: the oracle, as it stands, on the host cores, bounded sample ----
    cores = len(os.sched_getaffinity(0))
    n_cpu = oracle_requests_per_pass(w, keybits, cores, 1, budget_s=25.0)   # the same rule as the reference arm
    sample = oracle_sample(w, n_cpu)
    gbs, dt = oracle_throughput(w, keybits, n_cpu, cores, sample)
    n_one = max(1, min(n_cpu, int(4.0 * gbs / cores * 1e9 / size)))          # about 4 s on one core
    gbs1, dt1 = oracle_throughput(w, keybits, n_one, 1, sample)
    res["cpu_baseline"] = {"value": gbs, "unit": UNIT, "cores": cores, "kind": "oracle",
                           "sample": "%s %d of %d requests of %s (%d MiB), one thread per core, %.1f s" % (
                               "all" if n_cpu == n else "first", n_cpu, n, w.name, n_cpu * size // MIB, dt),
                           "one_core": {"value": gbs1, "unit": UNIT, "cores": 1,
                                        "sample": "first %d requests (%d MiB), %.1f s" % (n_one, n_one * size // MIB, dt1)}}
    res["cpu_context_aesni"] = openssl_speed(keybits)
    res["cpu_context_aesni_all_cores"] = openssl_speed(keybits, cores)
    return res


def openssl_speed(keybits, procs=1):
    """Context lines: OpenSSL's AES-NI/VAES CTR on ONE host core and on all of them, because the
    paper itself notes that 'a modern core's AES-NI rivals a GPU on this cipher'.  A fair "speed-up over the
    host" divides by THESE figures, not by the byte-wise oracle's.  Not a target."""
    import re
    import shutil
    import subprocess

    exe = shutil.which("openssl")
    if not exe:
        return {"unavailable": "no openssl binary on this box"}
    try:
        cmd = [exe, "speed", "-elapsed", "-evp", "aes-%d-ctr" % keybits, "-bytes", "1048576", "-seconds", "1"]
        if procs > 1:
            cmd += ["-multi", str(procs)]
        out = subprocess.run(cmd, capture_output=True, text=True, timeout=60).stdout
        m = re.search(r"^AES-%d-CTR\s+([0-9.]+)k" % keybits, out, re.M | re.I)
        if not m:
            return {"unavailable": "could not parse openssl speed output"}
        return {"value": float(m.group(1)) * 1000.0 / 1e9, "unit": UNIT, "cores": procs,
                "kind": "openssl speed -evp aes-%d-ctr%s, 1 MiB blocks (AES-NI/VAES)" % (keybits, " -multi %d" % procs if procs > 1 else "")}
    except Exception as e:  # noqa: BLE001
        return {"unavailable": str(e)}


def pcie_roof(torch, dev, hsv, hdv, piece):
    """What the link gives the copy engines over the SAME pinned buffers the e2e leg uses: cudaMemcpyAsync in pieces of
    32 MiB (issued from Python: request-sized pieces would measure the interpreter), host->device on one stream and
    device->host on another, alone and both at once.
    The both-at-once rate per direction is the roof a kernel that reads and writes host memory can be held against."""
    try:
        nbytes = len(hsv)
        hs_t, hd_t = torch.from_numpy(hsv), torch.from_numpy(hdv)
        if not (hs_t.is_pinned() and hd_t.is_pinned()):
            return None
        d_in = torch.empty(nbytes, dtype=torch.uint8, device=dev)
        d_out = torch.empty(nbytes, dtype=torch.uint8, device=dev)
        s_in, s_out = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
        torch.cuda.synchronize()

        def run(h2d, d2h, reps=3):
            best = None
            for _ in range(reps + 1):
                a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a0.record(s_in)
                b0.record(s_out)
                for off in range(0, nbytes, piece):
                    if h2d:
                        with torch.cuda.stream(s_in):
                            d_in[off:off + piece].copy_(hs_t[off:off + piece], non_blocking=True)
                    if d2h:
                        with torch.cuda.stream(s_out):
                            hd_t[off:off + piece].copy_(d_out[off:off + piece], non_blocking=True)
                a1.record(s_in)
                b1.record(s_out)
                torch.cuda.synchronize()
                ms = max(a0.elapsed_time(a1) if h2d else 0.0, b0.elapsed_time(b1) if d2h else 0.0)
                best = ms if best is None else min(best, ms)   # a roof: the best the link did (first pass = warm-up)
            return nbytes / (best * 1e-3) / 1e9

        return {"h2d_alone_gbs": run(True, False), "d2h_alone_gbs": run(False, True), "both_ways_gbs_each": run(True, True),
                "how": "copy engines, cudaMemcpyAsync per %d-byte piece over the e2e leg's own pinned buffers (%d MiB each way), "
                       "H2D and D2H on two streams at once, best of 3 after a warm-up pass, CUDA events" % (piece, nbytes // MIB)}
    except Exception as e:  # noqa: BLE001
        sys.stderr.write("pcie_roof: %s\n" % e)
        return None


if __name__ == "__main__":
    sys.exit(main())
