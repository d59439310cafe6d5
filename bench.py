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
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the launch backend, from the ncu --set full captures
# summarised in profiles/r1c_ncu.md (a persistent launch cannot be replayed by ncu)
NCU_TRAFFIC = {
    "c2": {"bytes": 67.25e6 + 25.27e6,
           "how": "ncu, one 64 x 1 MiB launch of the launch backend: 67.25 MB read + 25.27 MB written (algorithmic 67.11 + "
                  "67.11; the rest of the writes is still in the 126 MB L2 when the kernel ends); profiles/r1c_ncu.md"},
    "c3": {"bytes": 134.42e6 + 93.36e6,
           "how": "ncu, one 16 x 8 MiB launch of the launch backend: 134.42 MB read + 93.36 MB written (algorithmic 134.22 + "
                  "134.22); profiles/r1c_ncu.md"},
}
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
def oracle_throughput(w, keybits, n_req, cores):
    """Runs the oracle, as it stands, over the first n_req requests of w on `cores` threads.
    Returns (GB/s, seconds)."""
    import concurrent.futures as cf

    from oracle import oracle as o

    n_req = min(n_req, w.n)
    size = int(w.length[0])
    src = np.empty((n_req, size), dtype=np.uint8)
    dst = np.empty_like(src)
    for i in range(n_req):
        src[i] = w.payload(i)
    o.lib()

    def one(i):
        o.ctr_into(w.key_of(i), w.icb_of(i), src[i].ctypes.data, dst[i].ctypes.data, size)

    t0 = time.perf_counter()
    with cf.ThreadPoolExecutor(cores) as ex:
        list(ex.map(one, range(n_req)))
    dt = time.perf_counter() - t0
    return n_req * size / dt / 1e9, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w, keybits = make_workload(args.workload)
    cores = len(os.sched_getaffinity(0))
    per_step = max(cores, 16)  # requests per step: a bounded sample of the workload
    for _ in range(args.warmup):
        oracle_throughput(w, keybits, min(per_step, cores), cores)
    t_total, b_total = 0.0, 0
    for _ in range(args.steps):
        gbs, dt = oracle_throughput(w, keybits, per_step, cores)
        t_total += dt
        b_total += per_step * int(w.length[0])
    value = b_total / t_total / 1e9
    sample = "%d of the %d requests of %s per step (%d MiB), %d threads" % (
        per_step, w.n, w.name, per_step * int(w.length[0]) // MIB, cores)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps,
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
    ap.add_argument("--launch-requests", type=int, default=0,
                    help="--backend launch: requests per ordinary launch (0 = the config's in-flight window; the whole "
                         "batch in ONE launch is the operating point the ncu captures under profiles/ are made at)")
    ap.add_argument("--no-extras", action="store_true", help="skip e2e / latency / cpu_baseline / kernel-only legs")
    ap.add_argument("--sweep", action="store_true", help="configs[4]: size x in-flight x key-size table (one GPU)")
    ap.add_argument("--sweep-out", default="", help="with --sweep / --openloop: also write the table to this JSON file")
    ap.add_argument("--openloop", action="store_true", help="latency under Poisson load, blocking vs overlapping (PAPER.md:244)")
    ap.add_argument("--openloop-bytes", type=int, default=4096)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    if args.openloop:
        return run_openloop(args)
    if args.warmup < 3:
        args.warmup = 3

    import torch
    import torch.distributed as dist

    import paper_2607_02630_b200.binding as B
    from paper_2607_02630_b200 import multi

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
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

    def step_engine():
        r = B.aes_loop_run(w.icb, srcs, dsts, lens, window=w.in_flight, ctx=ctx, want_latency=False)
        assert r["requests"] == n

    LB = args.launch_requests or w.in_flight  # requests per ordinary launch in the launch backend

    def step_launch(stream_ptr, events=None):
        for b0 in range(0, n, LB):
            b1 = min(n, b0 + LB)
            if events is not None:
                e0 = torch.cuda.Event(enable_timing=True)
                e0.record()
            B.aes_ctr_launch_batch([ctx] * (b1 - b0), w.icb[b0:b1], srcs[b0:b1], dsts[b0:b1], lens[b0:b1],
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
                step_engine()
            ev1.record(side)
            side.synchronize()
            t1h = time.perf_counter()
            B.aes_engine_stop()
        else:
            ev0.record()
            for _ in range(args.steps):
                step_launch(torch.cuda.current_stream().cuda_stream, kernel_events)
            ev1.record()
        torch.cuda.synchronize()
        t1 = time.perf_counter() if args.backend != "engine" else t1h
    barrier()
    gpu_launches = B.aes_engine_info()["kernel_launches"] - launches_before
    ms_dev = ev0.elapsed_time(ev1)
    ms_host = 1e3 * (t1 - t0)
    # replicas only: every rank ran the same batch on its own engine; the job
    # took as long as its slowest rank
    bps, ms_total = multi.job_throughput(ms_dev, n * size * args.steps, dist if world > 1 else None, host_pg)
    value = bps / 1e9
    clk = clocks.summary()

    # ---- parity spot check of what the timed region wrote (rank 0; oracle is test infrastructure) ----
    verified = None
    if rank == 0:
        from oracle import oracle as o

        ok = True
        for i in (0, n // 2, n - 1):
            got = dst[i * size:i * size + 8192].cpu().numpy().tobytes()
            ok &= got == o.ctr(w.key_of(i), w.icb_of(i), w.payload(i)[:8192])
            off = size - 4096
            got = dst[i * size + off:(i + 1) * size].cpu().numpy().tobytes()
            ok &= got == o.ctr(w.key_of(i), w.icb_of(i), w.payload(i)[off:], off // 16)
        verified = bool(ok)

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
        "traffic": NCU_TRAFFIC.get(args.workload, {}).get("bytes"), "traffic_how": NCU_TRAFFIC.get(args.workload, {}).get("how"),
        "avg_launch_ms": kernel_ms, "how": how,
    }

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u8", "data": "synthetic",
        "config": {"workload": w.name, "backend": args.backend, "keybits": keybits, "request_bytes": size,
                   "requests_per_step": n, "in_flight": w.in_flight, "payload": "device-resident (HBM)",
                   "l2": "inputs larger than L2 (%.1f GiB src + same dst per step)" % (n * size / 2**30),
                   "seed": workloads.SEED_BASE + w.config_index},
        "gpu_launches": int(gpu_launches), "ms_host": ms_host, "engine_start_ms": engine_start_ms,
        "verified_vs_oracle": verified,
        "clocks": clk, "roofline": roofline,
    }

    if not args.no_extras and rank == 0 and world == 1:
        out.update(extras(args, B, torch, dev, local_rank, w, keybits, ctx, srcs, dsts, lens, size, n, step_launch,
                          lds_per_payload_byte, lds_peak, hbm_peak))
    elif rank == 0:
        out["e2e"] = None
    if rank == 0:
        print(json.dumps(out))
    B.aes_ctx_destroy(ctx)
    if world > 1:
        dist.destroy_process_group()
    return 0


def mix_c4(B, torch, dev, n=10000):
    """BASELINE.json configs[3] on the running engine: 10,000 requests, sizes log-uniform 1-64 KiB with
    0-15 B tails, a fresh AES-128 or AES-256 key per request (aes_ctx_create inside the timed loop; the raw
    key rides in the descriptor and is expanded by the dispatcher warp), random ICBs, 256 in flight."""
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
    B.aes_loop_run(w4.icb, srcs, dsts, w4.length, window=w4.in_flight, keys=keys, keybits=kb, want_latency=False)
    r = B.aes_loop_run(w4.icb, srcs, dsts, w4.length, window=w4.in_flight, keys=keys, keybits=kb)
    a = r["lat_ns"][n // 20:] / 1e3
    return {"workload": w4.name, "requests": n, "in_flight": w4.in_flight, "mean_bytes": float(w4.length.mean()),
            "p50_us": percentile(a, 50), "p99_us": percentile(a, 99), "req_per_s": n / (r["elapsed_ns"] * 1e-9),
            "payload_gbs": r["bytes"] / r["elapsed_ns"], "key_expansion": "per request, on the device"}


def run_sweep(args):
    """BASELINE.json configs[4]: payload 1 KiB .. 64 MiB in powers of two x in-flight 1/16/256/1024, AES-128 and
    AES-256, on the persistent engine; one JSON object per cell to stdout (and --sweep-out)."""
    import torch

    import paper_2607_02630_b200.binding as B

    hbm_peak, sm_max_mhz, _ = _peaks()
    dev = torch.device("cuda", 0)
    total = 8 << 30
    buf = torch.empty(total, dtype=torch.uint8, device=dev)
    buf.random_(0, 256)
    torch.cuda.synchronize()
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    lds_peak = SMEM_BYTES_PER_CLK_PER_SM * sm_count * sm_max_mhz * 1e6 / 1e9
    rng = np.random.Generator(np.random.Philox(key=[workloads.SEED_BASE + 5, 1]))
    cells = []
    B.aes_engine_start(0, idle_exit_ms=30000)
    try:
        for keybits in (128, 256):
            ctx = B.aes_ctx_create(rng.bytes(keybits // 8))
            for lg in range(10, 27):
                size = 1 << lg
                for depth in (1, 16, 256, 1024):
                    # distinct buffers while they fit; in place (dst == src) so that depth x size stays within `total`
                    nbuf = max(1, min(total // size, max(depth, 64)))
                    if nbuf < depth:
                        continue  # 64 MiB x 256 and up do not fit 8 GiB: cell skipped, stated in the output
                    # about 50 ms of work per cell, from a rough rate estimate
                    rate = min(600e9 / size, 4e6, depth / 10e-6)
                    n = int(min(max(0.05 * rate, 4 * depth, 64), 400000))
                    ptrs = np.asarray([buf.data_ptr() + (i % nbuf) * size for i in range(n)], dtype=np.uint64)
                    icb = np.zeros((n, 16), dtype=np.uint8)
                    icb[:, :8] = rng.integers(0, 256, size=(n, 8), dtype=np.uint8)
                    lens = np.full(n, size, dtype=np.uint64)
                    B.aes_loop_run(icb[:depth * 2], ptrs[:depth * 2], ptrs[:depth * 2], lens[:depth * 2], window=depth,
                                   ctx=ctx, want_latency=False)
                    r = B.aes_loop_run(icb, ptrs, ptrs, lens, window=depth, ctx=ctx)
                    a = r["lat_ns"][n // 20:] / 1e3
                    gbs = r["bytes"] / r["elapsed_ns"]
                    cell = {"keybits": keybits, "bytes": size, "in_flight": depth, "requests": n, "in_place": True,
                            "payload_gbs": gbs, "req_per_s": n / (r["elapsed_ns"] * 1e-9),
                            "p50_us": percentile(a, 50), "p99_us": percentile(a, 99),
                            "frac_lookup_roof": gbs * LOOKUPS[keybits] * 4.0 / 16.0 / lds_peak,
                            "frac_hbm_roof": 2 * gbs / hbm_peak}
                    cells.append(cell)
                    print(json.dumps(cell), flush=True)
            B.aes_ctx_destroy(ctx)
    finally:
        B.aes_engine_stop()
    if args.sweep_out:
        with open(args.sweep_out, "w") as f:
            json.dump({"lookup_roof_gbs_of_lookup_bytes": lds_peak, "hbm_peak_gbs": hbm_peak, "sm_mhz_assumed": sm_max_mhz,
                       "note": "in place; 64 MiB x 256/1024 in flight skipped (needs more than the 8 GiB the sweep allocates)",
                       "cells": cells}, f, indent=1)
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

    # ---- e2e: payloads in pinned HOST memory, read and written by the kernel over PCIe ----
    n_e2e = min(n, 256)
    hs = B.aes_host_alloc(n_e2e * size)
    hd = B.aes_host_alloc(n_e2e * size)
    hsv, hdv = B.host_view(hs, n_e2e * size), B.host_view(hd, n_e2e * size)
    for i in range(n_e2e):
        hsv[i * size:(i + 1) * size] = w.payload(i)
    hdv[:] = 0
    hsrcs = [hs + i * size for i in range(n_e2e)]
    hdsts = [hd + i * size for i in range(n_e2e)]
    B.aes_engine_start(local_rank, chunk_rows=args.chunk_rows, idle_exit_ms=30000)
    B.aes_loop_run(w.icb[:n_e2e], hsrcs, hdsts, lens[:n_e2e], window=w.in_flight, ctx=ctx, want_latency=False)
    reps = 4
    t0 = time.perf_counter()
    r = B.aes_loop_run(w.icb[:n_e2e], hsrcs, hdsts, lens[:n_e2e], window=w.in_flight, ctx=ctx, repeat=reps,
                       want_latency=False)
    t1 = time.perf_counter()
    from oracle import oracle as o

    ok = hdv[:4096].tobytes() == o.ctr(w.key_of(0), w.icb_of(0), w.payload(0)[:4096])
    e2e_gbs = r["bytes"] / (t1 - t0) / 1e9
    res["e2e"] = {"value": e2e_gbs, "unit": UNIT, "h2d_bytes_per_step": n_e2e * size, "d2h_bytes_per_step": n_e2e * size,
                  "how": "aes_ctr_submit with src/dst in pinned host memory (aes_host_alloc): the kernel reads the "
                         "payload and writes the result over PCIe inside the timed region; %d requests x %d B, %d in "
                         "flight, %d repeats" % (n_e2e, size, w.in_flight, reps),
                  "verified_vs_oracle": bool(ok)}

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
    # ---- configs[3]: the fine-grained mix, per-request keys (key expansion on the path) ----
    res["mix_c4"] = mix_c4(B, torch, dev)
    B.aes_engine_stop()
    B.aes_host_free(hl)
    # freeing pinned memory synchronises the device, so only after the engine has stopped
    del hsv, hdv
    B.aes_host_free(hs)
    B.aes_host_free(hd)

    # ---- calibration: what the lookup pipe, the ALU pipe and the payload path deliver on this GPU ----
    try:
        cal = B.aes_calibrate(local_rank)
        cal["lookup_pipe_frac_of_nominal"] = cal["lookups_per_clk_per_sm"] / 32.0
        cal["main_round_frac_of_nominal"] = cal["round_lookups_per_clk_per_sm"] / 32.0
        cal["how"] = ("aes_calibrate: microkernels with the engine's table layout and launch shape; nominal = 32 lookups and "
                      "2 warp-wide ALU instructions per clock per SM (guides/B300_MICROARCH.md)")
        res["calibration"] = cal
    except Exception as e:  # noqa: BLE001
        res["calibration"] = {"error": str(e)}

    # ---- cpu_baseline: the oracle, as it stands, on the host cores, bounded sample ----
    cores = len(os.sched_getaffinity(0))
    n_cpu = min(n, 16 * cores)
    gbs, dt = oracle_throughput(w, keybits, n_cpu, cores)
    res["cpu_baseline"] = {"value": gbs, "unit": UNIT, "cores": cores, "kind": "oracle",
                           "sample": "first %d of %d requests of %s (%d MiB), one thread per core, %.1f s" % (
                               n_cpu, n, w.name, n_cpu * size // MIB, dt)}
    res["cpu_context_aesni"] = openssl_speed(keybits)
    return res


def openssl_speed(keybits):
    """Second context line: OpenSSL's AES-NI/VAES CTR on ONE host core, because the paper
    itself notes that 'a modern core's AES-NI rivals a GPU on this cipher'.  Not a target."""
    import re
    import shutil
    import subprocess

    exe = shutil.which("openssl")
    if not exe:
        return {"unavailable": "no openssl binary on this box"}
    try:
        out = subprocess.run([exe, "speed", "-elapsed", "-evp", "aes-%d-ctr" % keybits, "-bytes", "1048576", "-seconds", "1"],
                             capture_output=True, text=True, timeout=30).stdout
        m = re.search(r"^AES-%d-CTR\s+([0-9.]+)k" % keybits, out, re.M | re.I)
        if not m:
            return {"unavailable": "could not parse openssl speed output"}
        return {"value": float(m.group(1)) * 1000.0 / 1e9, "unit": UNIT, "cores": 1,
                "kind": "openssl speed -evp aes-%d-ctr, 1 MiB blocks (AES-NI/VAES)" % keybits}
    except Exception as e:  # noqa: BLE001
        return {"unavailable": str(e)}


if __name__ == "__main__":
    sys.exit(main())
