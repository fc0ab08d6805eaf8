#!/usr/bin/env python
"""bench.py — pooled KV retrieve GB/s at 128K context on B200 (BASELINE.json metric).

    python bench.py --gpus N --steps K --warmup W            # the CUDA path (libkvpool.so through the C ABI)
    python bench.py --impl reference ...                     # the CPU oracle, as it stands, on the host cores

One STEP = one pass of the whole hot path over one request of the workload:
    kvpool_place  ->  kvpool_offload of every layer  ->  kvpool_retrieve of every layer (into a second paged pool)
The headline `value` is the retrieve leg: bytes moved by the retrieves of the K timed steps / their device time
(CUDA events on the launching stream, max over ranks).  `ms_per_step` is the whole step.  `e2e` is the same
retrieve leg by host wall clock through the public API, including the upload of the block tables from pinned
host memory, the host->GPU payload itself and a device->host read-back of one block per layer.

Prints ONE JSON line on stdout (rank 0).  Everything else goes to stderr / --detail.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "pooled_kv_retrieve_gbps_128k"
UNIT = "GB/s"
HBM_PEAK_FALLBACK = 6650.0      # GB/s, B200_PROFILING.md fallback ("of fallback") when MEASURED_PEAKS.json is absent


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["kvpool", "reference"], default="kvpool")
    ap.add_argument("--config", type=int, default=4, help="workload: 1..5 = BASELINE.json configs[0..4], 6 = LLaMA-8B alone at 128K")
    ap.add_argument("--path", choices=["auto", "staged", "zerocopy"], default="auto")
    ap.add_argument("--kernel", choices=["vec16", "bulk"], default=None)
    ap.add_argument("--weights", choices=["config", "measured", "equal"], default="config",
                    help="config: the weights BASELINE.json gives (measured where it gives none)")
    ap.add_argument("--link-ctas", type=int, default=0)
    ap.add_argument("--hbm-ctas", type=int, default=0)
    ap.add_argument("--stage-slots", type=int, default=0)
    ap.add_argument("--stage-chunk-mib", type=float, default=0.0,
                    help="staged path: cap a staging slot at this many MiB; larger layers travel in chunks (tune.stage_chunk_bytes)")
    ap.add_argument("--link-groups", choices=["shared", "independent"], default="shared",
                    help="shared (default): every host pool buffer names link group 1 - they all sit behind this GPU's one PCIe link, so the "
                         "library serves them in request order on one I/O stream per direction; independent: link group 0, one I/O stream "
                         "pair per pool device (the paper's literal 'independent I/O streams', PAPER.md:177)")
    ap.add_argument("--per-layer", action="store_true",
                    help="issue one kvpool_offload / kvpool_retrieve call per layer in the timed step instead of the batched *_layers calls")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--settle-s", type=float, default=60.0, help="upper bound on the untimed host-settle phase before the timed steps (0 = off)")
    ap.add_argument("--sweep", choices=["hbm", "link"], default=None,
                    help="tuning sweep instead of the benchmark: in-device pack/unpack (hbm) or zero-copy transfer (link) GB/s over launch shapes")
    ap.add_argument("--variants", action="store_true",
                    help="time the transfer variants side by side on --config (default 2): per-block cudaMemcpyAsync, staged, zero-copy")
    ap.add_argument("--blocked-io", action="store_true",
                    help="blocked-I/O-time analog (PAPER.md:70-72, Fig. 2/4): retrieve + consumer stand-in per layer, serial vs layerwise "
                         "pipelined, over context lengths 1K..128K for the three model shapes")
    ap.add_argument("--mixed-pool", action="store_true",
                    help="HBM-type pool devices (KVPOOL_DEV_HBM; the pool's own GPU standing in for an NVLink peer) next to a pinned "
                         "host device: bandwidth-proportional split by measured weights, offload / retrieve GB/s (DESIGN.md §11)")
    ap.add_argument("--duplex", action="store_true",
                    help="offload of one request concurrent with retrieve of another (PCIe is full duplex): per-direction and aggregate "
                         "GB/s against simultaneous cudaMemcpyAsync in both directions")
    ap.add_argument("--hostalloc", action="store_true", help="pool buffers from cudaHostAlloc (KVPOOL_DEV_CUDA_HOSTALLOC) instead of the default "
                    "huge-page mapping + cudaHostRegister; main run and --duplex")
    ap.add_argument("--compute-us", type=float, default=0.0, help="--blocked-io: extra calibrated compute per layer (kvpool_spin), microseconds")
    ap.add_argument("--detail", default=None, help="write per-layer latencies and side measurements to this JSON file")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks line")
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu, self.rows, self.proc, self.thread = gpu_index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        inside = [r for t, r in self.rows if t0 <= t <= t1] or [r for _, r in self.rows]
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in inside:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "source": "MEASURED_PEAKS.json (measured)"}
    return {"hbm_gbs": HBM_PEAK_FALLBACK, "source": "B200_PROFILING.md fallback"}


# ---------------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline of the kvpool arm; the whole of --impl reference)
# ---------------------------------------------------------------------------------------------------
def oracle_setup(cfg: int):
    """One layer of the workload on the host + the oracle's placement for it."""
    import oracle
    from paper_2606_14779_b200 import workloads as W
    wl = W.make_workload(cfg)
    bw = list(wl.default_weights())
    layer = max(range(wl.geom.n_layers), key=lambda l: wl.layer_span(0, l)[1])      # a full (non sliding-window) layer
    req = len(wl.requests) - 1                                                      # the 128K request class
    table = wl.layer_table(req, layer)
    pl = oracle.place(bw, [len(table)])[0]
    src = W.kv_layer_numpy(wl, layer)
    dst = W.poison_numpy(src.shape)
    return oracle, wl, table, pl, src, dst, layer, req


def oracle_time_layers(st, n_layers: int, parallel: bool):
    """Run offload+retrieve of the sample layer n_layers times; return (offload s, retrieve s, bytes per leg)."""
    oracle, wl, table, pl, src, dst, _, _ = st
    t_off = t_ret = 0.0
    for _ in range(n_layers):
        t0 = time.perf_counter()
        stripes = oracle.offload_layer(src, table, pl, parallel=parallel)
        t1 = time.perf_counter()
        oracle.retrieve_layer(dst, table, pl, stripes, parallel=parallel)
        t2 = time.perf_counter()
        t_off += t1 - t0
        t_ret += t2 - t1
    return t_off, t_ret, n_layers * len(table) * wl.geom.payload


def cpu_baseline(cfg: int, budget_s: float = 12.0) -> dict:
    st = oracle_setup(cfg)
    wl = st[1]
    n_threads = wl.n_pool_devices
    oracle_time_layers(st, 1, True)                                                 # touch pages
    t_off1, t_ret1, b1 = oracle_time_layers(st, 1, False)
    done, t_off, t_ret, nbytes = 0, 0.0, 0.0, 0
    t_start = time.perf_counter()
    while done < wl.geom.n_layers and time.perf_counter() - t_start < budget_s:
        a, b, c = oracle_time_layers(st, 1, True)
        t_off, t_ret, nbytes, done = t_off + a, t_ret + b, nbytes + c, done + 1
    return {"value": nbytes / t_ret / 1e9, "unit": UNIT, "cores": n_threads, "kind": "oracle",
            "sample": f"{done} x retrieve of one full layer of config {cfg} ({nbytes / done / 2**20:.0f} MiB each, host paged copy <- host stripes), "
                      f"one worker thread per pool device (PAPER.md:177); offload {nbytes / t_off / 1e9:.2f} GB/s; "
                      f"single-thread retrieve {b1 / t_ret1 / 1e9:.2f} GB/s",
            "host_cores": len(os.sched_getaffinity(0))}


def run_reference(args) -> dict:
    """--impl reference: the oracle as it stands on the host cores; a step = a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        sys.exit(0)
    st = oracle_setup(args.config)
    wl = st[1]
    layers_per_step = 4
    for _ in range(args.warmup):
        oracle_time_layers(st, 1, True)
    t_ret = t_all = 0.0
    nbytes = 0
    for _ in range(args.steps):
        a, b, c = oracle_time_layers(st, layers_per_step, True)
        t_ret, t_all, nbytes = t_ret + b, t_all + a + b, nbytes + c
    value = nbytes / t_ret / 1e9
    sample = (f"each step = offload+retrieve of {layers_per_step} full layers of config {args.config} "
              f"({nbytes / args.steps / 2**20:.0f} MiB per leg per step) on host memory")
    return {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_all / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8",
            "data": "synthetic", "config": {"workload": wl.name, "cfg": args.config, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": wl.n_pool_devices, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}


# ---------------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------------
def run_kvpool(args) -> dict:
    import torch
    from paper_2606_14779_b200 import binding as kv
    from paper_2606_14779_b200 import workloads as W

    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the kvpool arm has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    if not os.path.exists(kv.LIB_PATH):
        from paper_2606_14779_b200 import build as kvbuild
        kvbuild.build()
    kv.lib()

    wl = W.make_workload(args.config)
    g = wl.geom
    R, L, N = len(wl.requests), g.n_layers, wl.n_pool_devices
    elems = g.kvb // 2
    moved = wl.moved_bytes()
    bpl = [wl.blocks_per_layer(r) for r in range(R)]

    # ---- host-link peak of this box, measured now: 1 GiB pinned cudaMemcpyAsync, both directions ----
    probe = kv.KvPool([1.0], [1 << 30], n_layers=1, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim)
    link_h2d = max(probe.measure_bandwidth(0, 0, 1 << 30, 5) for _ in range(2))
    link_d2h = max(probe.measure_bandwidth(0, 1, 1 << 30, 5) for _ in range(2))
    probe.destroy()
    log(f"[rank {rank}] host link peak: H2D {link_h2d:.2f} GB/s, D2H {link_d2h:.2f} GB/s")

    # ---- the pool -------------------------------------------------------------------------------------------------
    base_w = list(wl.default_weights())
    share = np.array(base_w) / np.sum(base_w)
    caps = [int(moved * s * 1.25) + (L * R + 4) * (g.payload + 4096) for s in share]
    numa = [i % 2 for i in range(N)] if args.config == 2 else None      # config 2: "on 2 NUMA nodes" (falls back, reported)
    if numa is None and world > 1:
        numa = [kv.NUMA_AUTO] * N       # several ranks on one host: each rank's buffers on the NUMA node its own GPU hangs off
    t0 = time.perf_counter()
    pool = kv.KvPool(base_w, caps, n_layers=L, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim, block_tokens=g.block_tokens,
                     elem_bytes=g.elem_bytes, cuda_device=local, numa_nodes=numa,
                     dev_flags=[kv.DEV_CUDA_HOSTALLOC] * N if args.hostalloc else None,
                     link_groups=[1] * N if args.link_groups == "shared" else None)
    create_s = time.perf_counter() - t0
    weights_kind = args.weights
    if args.weights == "measured" or (args.weights == "config" and wl.weights is None):
        bw = [pool.measure_bandwidth(i, 0, min(256 << 20, caps[i]), 5) for i in range(N)]
        pool.set_bandwidth(bw)
        weights_kind = "measured per-buffer H2D GB/s"
    elif args.weights == "equal":
        bw = [1.0] * N
        pool.set_bandwidth(bw)
    else:
        bw = base_w
    pool.set_path({"auto": kv.PATH_AUTO, "staged": kv.PATH_STAGED, "zerocopy": kv.PATH_ZEROCOPY}[args.path])
    tune = {}
    if args.kernel:
        tune["kernel"] = tune["link_kernel"] = {"vec16": kv.KERNEL_VEC16, "bulk": kv.KERNEL_BULK}[args.kernel]
    for k, v in (("link_ctas", args.link_ctas), ("hbm_ctas", args.hbm_ctas), ("stage_slots", args.stage_slots)):
        if v:
            tune[k] = v
    if args.stage_chunk_mib:
        tune["stage_chunk_bytes"] = int(args.stage_chunk_mib * 2**20)
    if tune:
        pool.set_tuning(**tune)
    tn = pool.get_tuning()
    numa_actual = [pool.device_info(i)["numa_node"] for i in range(N)]
    log(f"[rank {rank}] pool: {N} buffers, {sum(caps) / 2**30:.1f} GiB pinned in {create_s:.1f} s, NUMA nodes {numa_actual}, weights {list(pool.weights())}")

    # ---- synthetic paged KV in HBM: source layers (seeded N(0,1) bf16) and poison-filled destination layers ---------
    src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
    dst = [W.poison_torch((2, wl.nphys, elems), dev) for l in range(L)]
    tables_np = [[np.ascontiguousarray(wl.layer_table(r, l)) for l in range(L)] for r in range(R)]
    tables_pin = [[torch.from_numpy(t).pin_memory() for t in row] for row in tables_np]
    tables = [[t.to(dev) for t in row] for row in tables_pin]
    table_bytes = sum(t.nbytes for row in tables_np for t in row)
    sample_pin = torch.empty((R, L, elems), dtype=torch.int16).pin_memory()
    main = torch.cuda.Stream(device=dev)
    streams = [torch.cuda.Stream(device=dev) for _ in range(max(1, wl.n_streams))] if wl.n_streams > 1 else [main]
    torch.cuda.synchronize()

    def fork():
        if streams[0] is not main:
            e = torch.cuda.Event()
            e.record(main)
            for s in streams:
                s.wait_event(e)

    def join():
        if streams[0] is not main:
            for s in streams:
                e = torch.cuda.Event()
                e.record(s)
                main.wait_event(e)

    src_k, src_v = [x[0] for x in src], [x[1] for x in src]
    dst_k, dst_v = [x[0] for x in dst], [x[1] for x in dst]

    def do_offload(pls):
        fork()
        if args.per_layer:
            for l in range(L):
                for r in range(R):
                    pool.offload(pls[r], l, src[l][0], src[l][1], g.kvb, tables[r][l], streams[r % len(streams)])
        else:
            for r in range(R):
                pool.offload_layers(pls[r], 0, src_k, src_v, g.kvb, tables[r], streams[r % len(streams)])
        for r in range(R):
            pool.wait_offloads(pls[r], streams[r % len(streams)])
        join()

    def do_retrieve(pls, layer_events=None, upload_tables=False):
        fork()
        if layer_events is None and not upload_tables and not args.per_layer:
            for r in range(R):
                pool.retrieve_layers(pls[r], 0, dst_k, dst_v, g.kvb, tables[r], streams[r % len(streams)])
            join()
            return
        for l in range(L):
            for r in range(R):
                s = streams[r % len(streams)]
                if upload_tables:
                    with torch.cuda.stream(s):
                        tables[r][l].copy_(tables_pin[r][l], non_blocking=True)
                pool.retrieve(pls[r], l, dst[l][0], dst[l][1], g.kvb, tables[r][l], s)
                if layer_events is not None:
                    e = torch.cuda.Event(enable_timing=True)
                    e.record(s)
                    layer_events[r].append(e)
        join()

    def step(timed: bool, rec: dict):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        t0 = time.perf_counter()
        pls = [pool.place(bpl[r]) for r in range(R)]
        t1 = time.perf_counter()
        ev[0].record(main)
        do_offload(pls)
        ev[1].record(main)
        # the legs are timed apart: without this the retrieve's host->GPU copies (which may run ahead of the caller's
        # stream) would start under the tail of the offload leg and borrow the link's other direction
        main.synchronize()
        pool.synchronize()
        ev[2].record(main)
        do_retrieve(pls)
        ev[3].record(main)
        main.synchronize()
        for pl in pls:
            pl.release()
        if timed:
            rec["place_ms"].append(1e3 * (t1 - t0))
            rec["offload_ms"].append(ev[0].elapsed_time(ev[1]))
            rec["retrieve_ms"].append(ev[2].elapsed_time(ev[3]))

    rec = {"place_ms": [], "offload_ms": [], "retrieve_ms": []}
    warm = {"place_ms": [], "offload_ms": [], "retrieve_ms": []}
    for _ in range(args.warmup):
        step(True, warm)
    # Host settle (untimed, disclosed in the JSON): in the first minutes after a GPU VM boots, DMA over a multi-GiB pinned
    # working set — and plain CPU memcpy — run 10-50 % below their steady state on this pool of boxes (the 1 GiB link probe
    # does not show it).  If the last warm-up leg is well below the link peak measured a moment ago, keep stepping, for at
    # most --settle-s seconds, until it is not.  A box that never gets there is timed as it is.
    settle = {"extra_steps": 0, "seconds": 0.0}
    t_settle = time.perf_counter()
    want_gbps = 0.9 * min(link_h2d, 55.0) * (0.92 if args.path == "zerocopy" else 1.0)
    while (args.settle_s > 0 and moved >= (1 << 30) and warm["retrieve_ms"] and moved / (warm["retrieve_ms"][-1] * 1e6) < want_gbps
           and time.perf_counter() - t_settle < args.settle_s):
        step(True, warm)
        settle["extra_steps"] += 1
        settle["seconds"] = time.perf_counter() - t_settle

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    # ---- the timed region: exactly K steps ---------------------------------------------------------------------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    k0, m0 = pool.stats()
    pool.set_profiling(True)
    barrier()
    t_begin = time.perf_counter()
    for _ in range(args.steps):
        step(True, rec)
    barrier()
    t_end = time.perf_counter()
    pool.set_profiling(False)
    k1, m1 = pool.stats()
    clocks = sampler.stop(t_begin, t_end) if rank == 0 else None
    prof_clk = {kind: pool.profile_read_clock(kind) for kind in range(4)}
    prof = {kind: (v[0], v[2], v[4]) for kind, v in prof_clk.items()}
    # one more step, untimed, with the timing events recorded on the launching streams themselves (kvpool.h: such a record
    # holds its stream up for 25-47 us under a concurrent copy-engine transfer): reported beside the side-stream figure
    pool.set_profiling(kv.PROFILE_INSTREAM)
    step(True, {"place_ms": [], "offload_ms": [], "retrieve_ms": []})
    pool.set_profiling(False)
    prof_in = {kind: pool.profile_read_clock(kind) for kind in range(4)}
    for kind, name in enumerate(("pack", "unpack", "zero-copy offload", "zero-copy retrieve")):
        if prof_clk[kind][2]:
            a, b_ = prof_clk[kind], prof_in[kind]
            log(f"[rank {rank}] {name}: {a[2]} launches; mean per launch: side-stream events {1e3 * a[0] / a[2]:.1f} us, kernel clock "
                f"{1e3 * a[1] / max(a[3], 1):.1f} us; in-stream events (extra step) {1e3 * b_[0] / max(b_[2], 1):.1f} us, kernel clock {1e3 * b_[1] / max(b_[3], 1):.1f} us")

    step_ms = 1e3 * (t_end - t_begin) / args.steps
    ret_ms = sum(rec["retrieve_ms"]) / args.steps
    off_ms = sum(rec["offload_ms"]) / args.steps
    if world > 1:
        import torch.distributed as dist
        t = torch.tensor([step_ms, ret_ms, off_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        step_ms, ret_ms, off_ms = [float(x) for x in t.tolist()]
    value = world * moved / (ret_ms * 1e6)

    # ---- correctness of what was timed: round trip bit-identical, nothing else written ---------------------------------
    verified = True
    for l in range(L):
        used = torch.zeros(wl.nphys, dtype=torch.bool, device=dev)
        for r in range(R):
            used[tables[r][l].long()] = True
        verified &= bool(torch.equal(dst[l][:, used], src[l][:, used]))
        verified &= bool((dst[l][:, ~used] == dst[l].new_tensor(np.int16(np.uint16(W.POISON_BITS).view(np.int16)).item())).all())
    if not verified:
        raise RuntimeError("retrieved KV differs from the source — refusing to report a number")

    # ---- e2e: the retrieve leg by host wall clock through the public API, tables uploaded from pinned host memory ------
    e2e_ret_s, e2e_off_s, layer_ms = [], [], [[] for _ in range(R)]
    for it in range(max(2, args.steps)):
        pls = [pool.place(bpl[r]) for r in range(R)]
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        do_offload(pls)
        main.synchronize()
        t1 = time.perf_counter()
        evs = [[] for _ in range(R)]
        start = torch.cuda.Event(enable_timing=True)
        start.record(main)
        do_retrieve(pls, layer_events=evs, upload_tables=True)
        with torch.cuda.stream(main):
            for r in range(R):
                for l in range(L):
                    if len(tables_np[r][l]):
                        sample_pin[r, l].copy_(dst[l][0, int(tables_np[r][l][0])], non_blocking=True)
        main.synchronize()
        t2 = time.perf_counter()
        for pl in pls:
            pl.release()
        if it > 0:                                          # first pass warms the pinned-table path
            e2e_off_s.append(t1 - t0)
            e2e_ret_s.append(t2 - t1)
            for r in range(R):
                prev = start
                for e in evs[r]:
                    layer_ms[r].append(prev.elapsed_time(e))
                    prev = e
    e2e_val = world * moved / (statistics.median(e2e_ret_s) * 1e9)
    d2h_bytes = sum(g.kvb for r in range(R) for l in range(L) if len(tables_np[r][l]))

    # ---- in-device pack / unpack alone (HBM roofline), rotating over layers so nothing is L2-resident ------------------
    hbm = {}
    big = max(range(L), key=lambda l: bpl[R - 1][l])
    Kbig = int(bpl[R - 1][big])
    pls = [pool.place(bpl[r]) for r in range(R)]
    stage = torch.empty(Kbig * g.payload, dtype=torch.uint8, device=dev)
    full_layers = [l for l in range(L) if int(bpl[R - 1][l]) == Kbig]
    for kname, kid in (("vec16", kv.KERNEL_VEC16), ("bulk", kv.KERNEL_BULK)):
        pool.set_tuning(kernel=kid)
        for op in ("pack", "unpack"):
            times = []
            for it in range(12):
                l = full_layers[it % len(full_layers)]
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(main)
                if op == "pack":
                    pool.pack(pls[R - 1], l, src[l][0], src[l][1], g.kvb, tables[R - 1][l], stage, main)
                else:
                    pool.unpack(pls[R - 1], l, dst[l][0], dst[l][1], g.kvb, tables[R - 1][l], stage, main)
                e1.record(main)
                main.synchronize()
                if it >= 2:
                    times.append(e0.elapsed_time(e1))
            hbm[f"{op}_{kname}_gbps"] = 2 * Kbig * g.payload / (statistics.median(times) * 1e6)
            # the same launches back to back (16 per event pair): amortises the ~10 us an event pair adds around one launch
            times = []
            for it in range(5):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(main)
                for i in range(16):
                    l = full_layers[i % len(full_layers)]
                    if op == "pack":
                        pool.pack(pls[R - 1], l, src[l][0], src[l][1], g.kvb, tables[R - 1][l], stage, main)
                    else:
                        pool.unpack(pls[R - 1], l, dst[l][0], dst[l][1], g.kvb, tables[R - 1][l], stage, main)
                e1.record(main)
                main.synchronize()
                if it >= 1:
                    times.append(e0.elapsed_time(e1) / 16)
            hbm[f"{op}_{kname}_back_to_back_gbps"] = 2 * Kbig * g.payload / (statistics.median(times) * 1e6)
    pool.set_tuning(kernel=tn.kernel)
    for pl in pls:
        pl.release()

    # ---- rooflines ---------------------------------------------------------------------------------------------------
    peaks = measured_peaks()
    kinds = ["pack (in-device)", "unpack (in-device)", "zero-copy offload", "zero-copy retrieve"]
    dom = max(range(4), key=lambda k: prof[k][0])
    ms, n, b = prof[dom]
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.csv")                            # ncu dram bytes per launch (profiles/traffic.md)
    if os.path.exists(tp):
        with open(tp) as f:
            for row in f.read().splitlines()[1:]:
                cfg, rest = row.split(",", 1)
                kind, nbytes = rest.rsplit(",", 1)
                if cfg == str(args.config) and kind == kinds[dom]:                  # captured per config; null where not captured
                    traffic = int(nbytes)
    if dom < 2:
        ach = 2 * b / (ms * 1e6) if ms > 0 else 0.0
        roof = {"bound": "hbm", "kernel": kinds[dom], "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
                "traffic": traffic, "peak_source": peaks["source"], "launches": n, "avg_launch_ms": ms / max(n, 1),
                "algorithmic_bytes_per_launch": 2 * b // max(n, 1), "frac_of_8TBs_nominal": ach / 8000.0}
        ims, _, inn, _, ib = prof_in[dom]
        if inn and ims > 0:
            roof.update({"achieved_instream_events": 2 * ib / (ims * 1e6), "frac_instream_events": 2 * ib / (ims * 1e6) / peaks["hbm_gbs"],
                         "avg_launch_ms_instream_events": ims / inn})
        roof["timing"] = ("CUDA timing events on two side streams of the pool, gated by non-timing marker events recorded on the launching "
                          "stream right before and right after the kernel (kvpool_set_profiling, KVPOOL_PROFILE_SIDE)")
        _, dms, _, nd, _ = prof_clk[dom]
        if nd:
            # the same launches of the timed region by the kernels' own clock (%globaltimer: first CTA start to last CTA end)
            clk = 2 * (b / n) * nd / (dms * 1e6)
            roof.update({"achieved_kernel_clock": clk, "frac_kernel_clock": clk / peaks["hbm_gbs"], "avg_launch_ms_kernel_clock": dms / nd,
                         "launches_kernel_clock": nd})
    else:
        peak = link_d2h if dom == 2 else link_h2d
        ach = b / (ms * 1e6) if ms > 0 else 0.0
        roof = {"bound": "host_link", "kernel": kinds[dom], "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": traffic,
                "peak_source": "1 GiB pinned cudaMemcpyAsync measured in this run", "launches": n, "avg_launch_ms": ms / max(n, 1),
                "algorithmic_bytes_per_launch": b // max(n, 1)}
    link_roof = {"bound": "host_link", "what": "retrieve leg (all layers back to back)", "achieved": value / world, "peak": link_h2d,
                 "unit": "GB/s", "frac": value / world / link_h2d, "offload_achieved": moved / (off_ms * 1e6), "offload_peak": link_d2h,
                 "offload_frac": moved / (off_ms * 1e6) / link_d2h, "peak_source": "1 GiB pinned cudaMemcpyAsync measured in this run"}
    best_unpack = max(hbm["unpack_vec16_back_to_back_gbps"], hbm["unpack_bulk_back_to_back_gbps"])
    best_pack = max(hbm["pack_vec16_back_to_back_gbps"], hbm["pack_bulk_back_to_back_gbps"])
    hbm_roof = {"bound": "hbm", "what": f"in-device pack/unpack of one {Kbig * g.payload / 2**20:.0f} MiB layer launched alone, 2*bytes/time; "
                "*_gbps = one launch per event pair, *_back_to_back_gbps = 16 launches per event pair", **hbm,
                "peak": peaks["hbm_gbs"], "frac_unpack": best_unpack / peaks["hbm_gbs"], "frac_pack": best_pack / peaks["hbm_gbs"],
                "frac_unpack_of_8TBs_nominal": best_unpack / 8000.0, "frac_pack_of_8TBs_nominal": best_pack / 8000.0}
    if dom < 2 and Kbig * g.payload >= (64 << 20):      # (a 4 MiB launch measures launch latency, not bandwidth: no reference then)
        # the measured peak's own kernel (a contiguous torch copy_ of the same bytes) under the in-step condition: a copy
        # engine streaming over the host link in the direction of that leg (offload: D2H, retrieve: H2D)
        side, big_d = torch.empty(Kbig * g.payload, dtype=torch.uint8, device=dev), torch.empty(1 << 30, dtype=torch.uint8, device=dev)
        big_h, other = torch.empty(1 << 30, dtype=torch.uint8).pin_memory(), torch.cuda.Stream(device=dev)

        def bg():
            with torch.cuda.stream(other):
                (big_h if dom == 0 else big_d).copy_(big_d if dom == 0 else big_h, non_blocking=True)

        def k_copy(i):
            with torch.cuda.stream(main):
                stage.copy_(side, non_blocking=True)

        ref_us = time_under_dma(torch, main, other, k_copy, bg)
        ref_alone_us = time_under_dma(torch, main, other, k_copy, None)
        roof["empty_event_pair_under_dma_us"] = time_under_dma(torch, main, other, lambda i: None, bg)
        roof["empty_event_pair_alone_us"] = time_under_dma(torch, main, other, lambda i: None, None)
        roof["torch_copy_same_bytes_under_dma_gbps"] = 2 * Kbig * g.payload / ref_us / 1e3
        roof["torch_copy_same_bytes_alone_gbps"] = 2 * Kbig * g.payload / ref_alone_us / 1e3
        roof["frac_of_torch_copy_under_dma"] = ach / roof["torch_copy_same_bytes_under_dma_gbps"]
        del side, big_d, big_h
    if dom < 2:
        kn = "vec16" if tn.kernel == kv.KERNEL_VEC16 else "bulk"
        roof["achieved_back_to_back"] = hbm[f"{'pack' if dom == 0 else 'unpack'}_{kn}_back_to_back_gbps"]
        roof["frac_back_to_back"] = roof["achieved_back_to_back"] / peaks["hbm_gbs"]
        roof["note"] = ("achieved = per-launch CUDA timing-event pairs inside the timed step, where every pack/unpack launch runs while the "
                        "copy engines stream the neighbouring layers over the host link; the events sit on side streams behind non-timing "
                        "markers (see timing) because a timing event recorded on the launching stream holds that stream up until its "
                        "timestamp is written - empty_event_pair_under_dma_us with nothing between the records, vs "
                        "empty_event_pair_alone_us - which delays the kernel and counts the delay: achieved_instream_events is that "
                        "measurement (one extra untimed step), and a plain torch copy_ of the same bytes timed that way pays the same "
                        "(torch_copy_same_bytes_under_dma_gbps; profiles/r1_interference.txt); "
                        "achieved_kernel_clock = the same in-step launches timed by the kernel itself (%globaltimer, first CTA start to "
                        "last CTA end, stores fenced); achieved_back_to_back = same kernel, 16 launches per event pair, no concurrent copy")

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": step_ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": wl.name, "cfg": args.config, "context_tokens": list(wl.context_tokens), "layers": L, "requests": R,
                   "moved_bytes_per_leg": moved, "pool_buffers": N, "weights": weights_kind, "bandwidth_gbps": [round(float(x), 3) for x in bw],
                   "numa_nodes": numa_actual, "path": args.path, "kernel": "vec16" if tn.kernel == kv.KERNEL_VEC16 else "bulk",
                   "link_kernel": "vec16" if tn.link_kernel == kv.KERNEL_VEC16 else "bulk",
                   "link_ctas": tn.link_ctas, "hbm_ctas": tn.hbm_ctas, "stage_slots": tn.stage_slots, "stage_chunk_bytes": tn.stage_chunk_bytes, "link_groups": args.link_groups, "streams": len(streams),
                   "l2": f"inputs larger than L2: each leg moves {moved / 2**30:.1f} GiB through {L} distinct layers (L2 is 126 MB); no flush needed",
                   "calls": "per-layer" if args.per_layer else "batched (kvpool_offload_layers / kvpool_retrieve_layers, one call per request)",
                   "step": "kvpool_place + offload of every layer + retrieve of every layer; value = retrieve leg"},
        "retrieve_ms_per_step": ret_ms, "offload_ms_per_step": off_ms, "offload_gbps": world * moved / (off_ms * 1e6),
        "place_ms_per_step": statistics.mean(rec["place_ms"]), "verified_bit_exact_round_trip": verified,
        "pool_create": {"seconds": create_s, "pinned_bytes": int(sum(caps)), "gbps": sum(caps) / create_s / 1e9,
                        "what": "kvpool_create: huge-page mapping faulted in by up to 16 threads + cudaHostRegister (outside the timed region)"},
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": moved + table_bytes, "d2h_bytes_per_step": d2h_bytes,
                "what": "retrieve leg by host wall clock: pinned block tables H2D + kvpool_retrieve x layers + D2H of one block per layer + sync",
                "offload_gbps": world * moved / (statistics.median(e2e_off_s) * 1e9)},
        "gpu_launches": k1 - k0, "memcpy_calls": m1 - m0, "host_settle": settle,
        "roofline": roof, "roofline_link": link_roof, "roofline_hbm": hbm_roof,
        "clocks": clocks,
    }
    per_layer = [x for r in range(R) for x in layer_ms[r]]
    if per_layer:
        per_layer.sort()
        out["retrieve_layer_ms"] = {"min": per_layer[0], "median": per_layer[len(per_layer) // 2], "p99": per_layer[min(len(per_layer) - 1, int(0.99 * len(per_layer)))],
                                    "what": "interval between consecutive per-layer completion events on a request's stream, retrieve leg"}
    if args.detail and rank == 0:
        with open(args.detail, "w") as f:
            json.dump({"out": out, "rec": rec, "layer_ms": layer_ms, "prof": {kinds[k]: prof[k] for k in range(4)}}, f, indent=1)
    pool.destroy()
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return out if rank == 0 else None


def run_sweep(args) -> None:
    """Tuning sweeps on a 4-layer cut of the workload (text table on stdout)."""
    import itertools
    import torch
    from paper_2606_14779_b200 import binding as kv
    from paper_2606_14779_b200 import workloads as W

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    wl = W.make_workload(args.config, n_layers=4)
    wl.sliding_layers = ()
    g, R = wl.geom, len(wl.requests) - 1
    bw = list(wl.default_weights())
    K = int(wl.blocks_per_layer(R)[0])
    share = np.array(bw) / np.sum(bw)
    caps = [int(wl.moved_bytes() * s * 1.25) + 64 * (g.payload + 4096) for s in share]
    pool = kv.KvPool(bw, caps, n_layers=4, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim)
    probe_h2d = pool.measure_bandwidth(0, 0, min(256 << 20, caps[0]), 5)
    probe_d2h = pool.measure_bandwidth(0, 1, min(256 << 20, caps[0]), 5)
    pl = pool.place(wl.blocks_per_layer(R))
    src = [W.kv_layer_torch(wl, l, dev) for l in range(4)]
    tables = [torch.from_numpy(np.ascontiguousarray(wl.layer_table(R, l))).to(dev) for l in range(4)]
    stage = torch.empty(K * g.payload, dtype=torch.uint8, device=dev)
    main_s = torch.cuda.Stream(device=dev)
    torch.cuda.synchronize()
    nbytes = K * g.payload

    def timed(fn, reps, per_pair):
        ts = []
        for it in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(main_s)
            for i in range(per_pair):
                fn((it * per_pair + i) % 4)
            e1.record(main_s)
            main_s.synchronize()
            if it >= 2:
                ts.append(e0.elapsed_time(e1) / per_pair)
        return statistics.median(ts)

    print(f"# bench.py --sweep {args.sweep} --config {args.config}: {wl.name}, K={K} blocks of P={g.payload} B = {nbytes / 2**20:.0f} MiB per launch")
    if args.sweep == "hbm":
        print("# in-device pack / unpack, GB/s = 2*bytes/time, 8 launches per event pair, median of 6; measured HBM copy peak "
              f"{measured_peaks()['hbm_gbs']:.0f} GB/s")
        for threads, unroll, ctas in itertools.product((128, 256, 512), (4, 8, 16), (148, 296, 592, 1184, 2368, 4736)):
            pool.set_tuning(kernel=kv.KERNEL_VEC16, vec_threads=threads, vec_unroll=unroll, hbm_ctas=ctas)
            p = timed(lambda l: pool.pack(pl, l, src[l][0], src[l][1], g.kvb, tables[l], stage, main_s), 8, 8)
            u = timed(lambda l: pool.unpack(pl, l, src[l][0], src[l][1], g.kvb, tables[l], stage, main_s), 8, 8)
            print(f"vec16 threads {threads:4d} unroll {unroll:2d} ctas {ctas:5d}: pack {2 * nbytes / p / 1e6:6.0f}  unpack {2 * nbytes / u / 1e6:6.0f}", flush=True)
        for warps, stages, chunk, ctas in [(1, 8, 16384, 148), (2, 6, 16384, 148), (2, 4, 16384, 148), (4, 6, 8192, 148), (4, 4, 8192, 296),
                                           (2, 3, 16384, 296), (2, 3, 32768, 148), (4, 3, 16384, 148), (8, 3, 8192, 148), (8, 6, 4096, 148)]:
            pool.set_tuning(kernel=kv.KERNEL_BULK, bulk_warps=warps, bulk_stages=stages, bulk_chunk=chunk, hbm_ctas=ctas)
            p = timed(lambda l: pool.pack(pl, l, src[l][0], src[l][1], g.kvb, tables[l], stage, main_s), 8, 8)
            u = timed(lambda l: pool.unpack(pl, l, src[l][0], src[l][1], g.kvb, tables[l], stage, main_s), 8, 8)
            print(f"bulk warps {warps} stages {stages} chunk {chunk:5d} ctas {ctas:4d}: pack {2 * nbytes / p / 1e6:6.0f}  unpack {2 * nbytes / u / 1e6:6.0f}", flush=True)
    else:
        print(f"# zero-copy offload / retrieve of one layer, GB/s = bytes/time, 1 launch per event pair, median of 4; cudaMemcpyAsync 256 MiB: "
              f"H2D {probe_h2d:.2f} D2H {probe_d2h:.2f} GB/s")
        pool.set_path(kv.PATH_ZEROCOPY)
        cases = [(kv.KERNEL_VEC16, "vec16", dict(vec_threads=t)) for t in (128, 256, 512)] + \
                [(kv.KERNEL_BULK, "bulk", dict(bulk_warps=w, bulk_stages=s_, bulk_chunk=c)) for w, s_, c in ((1, 4, 16384), (1, 8, 16384), (2, 6, 16384), (4, 6, 8192))]
        for kid, name, extra in cases:
            for ctas in (1, 2, 4, 8, 16, 32, 148):
                pool.set_tuning(link_kernel=kid, link_ctas=ctas, **extra)
                o = timed(lambda l: pool.offload(pl, l, src[l][0], src[l][1], g.kvb, tables[l], main_s), 6, 1)
                r = timed(lambda l: pool.retrieve(pl, l, src[l][0], src[l][1], g.kvb, tables[l], main_s), 6, 1)
                print(f"{name} {extra} ctas {ctas:4d}: offload {nbytes / o / 1e6:6.2f}  retrieve {nbytes / r / 1e6:6.2f}", flush=True)
    pl.release()
    pool.destroy()


def run_variants(args) -> None:
    """V0 per-block cudaMemcpyAsync (what an engine without a gather kernel does), V2 pack/unpack kernel + one
    cudaMemcpyAsync per stripe (the north star's baseline path), V3 zero-copy 16-byte vector kernel, V4 zero-copy
    cp.async.bulk kernel.  Whole request, per-layer calls, legs timed apart with CUDA events.  Text table on stdout."""
    import torch
    from paper_2606_14779_b200 import binding as kv
    from paper_2606_14779_b200 import workloads as W

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    cfg = args.config if args.config != 4 or "--config" in sys.argv else 2
    wl = W.make_workload(cfg)
    g, L = wl.geom, wl.geom.n_layers
    bw = list(wl.default_weights())
    share = np.array(bw) / np.sum(bw)
    moved = int(wl.blocks_per_layer(0).sum()) * g.payload
    caps = [int(moved * sh * 1.25) + (L + 4) * (g.payload + 4096) for sh in share]
    pool = kv.KvPool(bw, caps, n_layers=L, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim)
    h2d = pool.measure_bandwidth(0, 0, min(256 << 20, caps[0]), 5)
    d2h = pool.measure_bandwidth(0, 1, min(256 << 20, caps[0]), 5)
    bpl = wl.blocks_per_layer(0)
    elems = g.kvb // 2
    src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
    dst = [W.poison_torch((2, wl.nphys, elems), dev) for l in range(L)]
    tables_np = [np.ascontiguousarray(wl.layer_table(0, l)) for l in range(L)]
    tables = [torch.from_numpy(t).to(dev) for t in tables_np]
    s = torch.cuda.Stream(device=dev)
    torch.cuda.synchronize()
    print(f"# bench.py --variants --config {cfg}: {wl.name}, {moved / 2**20:.0f} MiB per leg over {L} layers, {wl.n_pool_devices} pool buffers; "
          f"cudaMemcpyAsync 256 MiB: H2D {h2d:.2f} D2H {d2h:.2f} GB/s; median of 3")
    print(f"{'variant':58s} {'offload GB/s':>12s} {'retrieve GB/s':>13s} {'x H2D peak':>10s} {'kernels':>8s} {'memcpys':>8s}")
    variants = [
        ("V0 per-block cudaMemcpyAsync (2*K_l calls per layer)", "naive", {}),
        ("V2 staged: vec16 pack/unpack + 1 memcpy per stripe", kv.PATH_STAGED, dict(kernel=kv.KERNEL_VEC16)),
        ("V2 staged: bulk pack/unpack + 1 memcpy per stripe", kv.PATH_STAGED, dict(kernel=kv.KERNEL_BULK)),
        ("V3 zero-copy vec16 kernel, 8 CTAs", kv.PATH_ZEROCOPY, dict(link_kernel=kv.KERNEL_VEC16, link_ctas=8)),
        ("V4 zero-copy cp.async.bulk kernel, 4 CTAs", kv.PATH_ZEROCOPY, dict(link_kernel=kv.KERNEL_BULK, link_ctas=4)),
        ("V4 zero-copy cp.async.bulk kernel, 2 CTAs", kv.PATH_ZEROCOPY, dict(link_kernel=kv.KERNEL_BULK, link_ctas=2)),
    ]
    for name, path, tune in variants:
        if path != "naive":
            pool.set_path(path)
            pool.set_tuning(**tune)
        offs, rets = [], []
        k0, m0 = pool.stats()
        for it in range(4):
            for d in dst:
                d.fill_(np.int16(np.uint16(W.POISON_BITS).view(np.int16)).item())
            pl = pool.place(bpl)
            torch.cuda.synchronize()
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            ev[0].record(s)
            for l in range(L):
                if path == "naive":
                    pool.offload_naive(pl, l, src[l][0], src[l][1], g.kvb, tables_np[l], s)
                else:
                    pool.offload(pl, l, src[l][0], src[l][1], g.kvb, tables[l], s)
            pool.wait_offloads(pl, s)
            ev[1].record(s)
            s.synchronize()
            pool.synchronize()
            ev[2].record(s)
            for l in range(L):
                if path == "naive":
                    pool.retrieve_naive(pl, l, dst[l][0], dst[l][1], g.kvb, tables_np[l], s)
                else:
                    pool.retrieve(pl, l, dst[l][0], dst[l][1], g.kvb, tables[l], s)
            ev[3].record(s)
            s.synchronize()
            pl.release()
            if it > 0:
                offs.append(ev[0].elapsed_time(ev[1]))
                rets.append(ev[2].elapsed_time(ev[3]))
        k1, m1 = pool.stats()
        for l in range(L):
            if not torch.equal(dst[l][:, tables[l].long()], src[l][:, tables[l].long()]):
                raise RuntimeError(f"{name}: retrieved KV differs from the source")
        o, r = moved / statistics.median(offs) / 1e6, moved / statistics.median(rets) / 1e6
        print(f"{name:58s} {o:12.2f} {r:13.2f} {r / h2d:10.3f} {(k1 - k0) // 4:8d} {(m1 - m0) // 4:8d}", flush=True)
    pool.destroy()


def time_under_dma(torch, s, o, fn, bg, launches: int = 16, reps: int = 4):
    """Median microseconds of fn(i) on stream `s`, one CUDA event pair per launch, while `bg()` (a long cudaMemcpyAsync
    enqueued on stream `o`; None = nothing) is in flight.  Best of reps-1 after one warm-up repetition."""
    best = None
    for rep in range(reps):
        torch.cuda.synchronize()
        if bg:
            bg()
            time.sleep(0.005)                # the background transfer is under way
        ts = []
        for i in range(launches):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(s)
            fn(i)
            e1.record(s)
            ts.append((e0, e1))
        s.synchronize()
        covered = bg is None or not o.query()
        torch.cuda.synchronize()
        if not covered:
            raise RuntimeError("the background transfer ended before the timed launches did")
        us = 1e3 * statistics.median(a.elapsed_time(b) for a, b in ts)
        if rep > 0:
            best = us if best is None else min(best, us)
    return best


def run_mixed_pool(args) -> None:
    """Eq. 1-2 at work on devices of very different speed: one pinned host buffer (PCIe) and one HBM-type device, alone and
    together, weights = kvpool_measure_bandwidth of each.  Whole request (16 layers of --config), batched calls, legs
    timed apart with CUDA events; every run is verified bit-exact against the source.  Text table on stdout."""
    import torch
    from paper_2606_14779_b200 import binding as kv
    from paper_2606_14779_b200 import workloads as W

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    L = 16
    wl = W.make_workload(args.config, n_layers=L)
    wl.sliding_layers = ()
    g = wl.geom
    bpl = wl.blocks_per_layer(0)
    K, moved = int(bpl[0]), int(bpl.sum()) * g.payload
    elems = g.kvb // 2
    src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
    dst = [W.poison_torch((2, wl.nphys, elems), dev) for l in range(L)]
    tables = [torch.from_numpy(np.ascontiguousarray(wl.layer_table(0, l))).to(dev) for l in range(L)]
    src_k, src_v, dst_k, dst_v = [x[0] for x in src], [x[1] for x in src], [x[0] for x in dst], [x[1] for x in dst]
    s = torch.cuda.Stream(device=dev)
    torch.cuda.synchronize()
    cap = moved + (L + 4) * (g.payload + 4096)
    print(f"# bench.py --mixed-pool --config {args.config}: {wl.name} cut to {L} layers, {moved / 2**20:.0f} MiB per leg ({K} blocks of {g.payload} B per layer); "
          "weights = kvpool_calibrate (256 MiB per device: cudaMemcpyAsync for the host-only pool, the gather kernel itself for pools with HBM-type devices; link groups "
          "share; payload GB/s); median of 3; HBM-type device = this GPU's own memory")
    print(f"{'pool':34s} {'weights (GB/s)':>22s} {'blocks per layer':>18s} {'offload GB/s':>12s} {'retrieve GB/s':>13s} {'sum of weights':>14s} {'kernels':>8s} {'memcpys':>8s}")
    for name, flags in (("1 host buffer", [0]), ("1 host buffer + 1 HBM device", [0, kv.DEV_HBM]), ("2 host buffers + 2 HBM devices", [0, 0, kv.DEV_HBM, kv.DEV_HBM]),
                        ("1 HBM device", [kv.DEV_HBM])):
        n = len(flags)
        # devices behind ONE shared resource name one link group (the host buffers behind this GPU's single PCIe link: 1; the
        # HBM-type devices inside one GPU: 2): kvpool_calibrate measures every device and divides what a group shares.  A pool
        # with HBM-type devices is measured with the library's own kernel, which is what reaches every stripe there.
        pool = kv.KvPool([1.0] * n, [cap] * n, n_layers=L, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim, dev_flags=flags,
                         link_groups=[2 if f else 1 for f in flags])
        bw = list(pool.calibrate(kv.MEASURE_KERNEL_RETRIEVE if any(flags) else kv.MEASURE_RETRIEVE, 256 << 20, 5))
        offs, rets = [], []
        k0, m0 = pool.stats()
        for it in range(4):
            for d in dst:
                d.fill_(np.int16(np.uint16(W.POISON_BITS).view(np.int16)).item())
            pl = pool.place(bpl)
            counts = list(pl.counts(0))
            torch.cuda.synchronize()
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            ev[0].record(s)
            pool.offload_layers(pl, 0, src_k, src_v, g.kvb, tables, s)
            pool.wait_offloads(pl, s)
            ev[1].record(s)
            s.synchronize()
            pool.synchronize()
            ev[2].record(s)
            pool.retrieve_layers(pl, 0, dst_k, dst_v, g.kvb, tables, s)
            ev[3].record(s)
            s.synchronize()
            pl.release()
            if it > 0:
                offs.append(ev[0].elapsed_time(ev[1]))
                rets.append(ev[2].elapsed_time(ev[3]))
        k1, m1 = pool.stats()
        for l in range(L):
            if not torch.equal(dst[l][:, tables[l].long()], src[l][:, tables[l].long()]):
                raise RuntimeError(f"{name}: retrieved KV differs from the source")
        o, r = moved / statistics.median(offs) / 1e6, moved / statistics.median(rets) / 1e6
        print(f"{name:34s} {'/'.join(f'{b:.0f}' for b in bw):>22s} {'/'.join(str(c) for c in counts):>18s} {o:12.1f} {r:13.1f} {sum(bw):14.0f} "
              f"{(k1 - k0) // 4:8d} {(m1 - m0) // 4:8d}", flush=True)
        pool.destroy()


def run_duplex(args) -> None:
    """A serving engine evicts one request's KV while it fetches another's.  Request A is offloaded on one stream while
    request B (offloaded beforehand) is retrieved on another; both legs are timed with CUDA events on their own stream and
    the pair by the wall clock.  Peak = two simultaneous 1 GiB pinned cudaMemcpyAsync, one per direction.  Text table."""
    import torch
    from paper_2606_14779_b200 import binding as kv
    from paper_2606_14779_b200 import workloads as W

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    L = 16
    wl = W.make_workload(args.config, n_layers=L)
    wl.sliding_layers = ()
    g = wl.geom
    bpl = wl.blocks_per_layer(0)
    moved = int(bpl.sum()) * g.payload
    elems = g.kvb // 2
    bw = list(wl.default_weights())
    share = np.array(bw) / np.sum(bw)
    caps = [int(2 * moved * sh * 1.25) + 2 * (L + 4) * (g.payload + 4096) for sh in share]
    pool = kv.KvPool(bw, caps, n_layers=L, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim,
                     dev_flags=[kv.DEV_CUDA_HOSTALLOC] * len(bw) if args.hostalloc else None)
    src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
    dst = [W.poison_torch((2, wl.nphys, elems), dev) for l in range(L)]
    tables = [torch.from_numpy(np.ascontiguousarray(wl.layer_table(0, l))).to(dev) for l in range(L)]
    src_k, src_v, dst_k, dst_v = [x[0] for x in src], [x[1] for x in src], [x[0] for x in dst], [x[1] for x in dst]
    sa, sb = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)

    # duplex peak of the link: simultaneous H2D and D2H copies of 1 GiB each
    hd, dd = torch.empty(1 << 30, dtype=torch.uint8).pin_memory(), torch.empty(1 << 30, dtype=torch.uint8, device=dev)
    hu, du = torch.empty(1 << 30, dtype=torch.uint8).pin_memory(), torch.empty(1 << 30, dtype=torch.uint8, device=dev)
    hd.copy_(dd)          # freshly zeroed host pages read slow over the link until a DMA write has claimed them
    peak = []
    for it in range(4):
        torch.cuda.synchronize()
        e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        with torch.cuda.stream(sa):
            e[0].record(sa); dd.copy_(hd, non_blocking=True); e[1].record(sa)
        with torch.cuda.stream(sb):
            e[2].record(sb); hu.copy_(du, non_blocking=True); e[3].record(sb)
        torch.cuda.synchronize()
        if it:
            peak.append(((1 << 30) / e[0].elapsed_time(e[1]) / 1e6, (1 << 30) / e[2].elapsed_time(e[3]) / 1e6))
    peak_h2d, peak_d2h = statistics.median(p[0] for p in peak), statistics.median(p[1] for p in peak)
    del hd, dd, hu, du
    torch.cuda.synchronize()
    print(f"# bench.py --duplex --config {args.config}: {wl.name} cut to {L} layers; request A ({moved / 2**20:.0f} MiB) is offloaded while request B "
          f"({moved / 2**20:.0f} MiB) is retrieved; median of 3")
    print(f"# simultaneous cudaMemcpyAsync, 1 GiB each way: H2D {peak_h2d:.1f} GB/s + D2H {peak_d2h:.1f} GB/s = {peak_h2d + peak_d2h:.1f} GB/s")
    print(f"{'path/CTAs':12s} {'offload A GB/s':>15s} {'retrieve B GB/s':>16s} {'aggregate GB/s (wall)':>22s} {'x duplex peak':>14s}")
    if args.stage_slots:
        pool.set_tuning(stage_slots=args.stage_slots)
    for pname, path, ctas in (("staged", kv.PATH_STAGED, 0), ("zerocopy", kv.PATH_ZEROCOPY, args.link_ctas or 4),
                              ("zerocopy", kv.PATH_ZEROCOPY, 4 * (args.link_ctas or 4))):
        pool.set_path(path)
        if ctas:
            pool.set_tuning(link_ctas=ctas)
            pname = f"{pname}/{ctas}"
        offs, rets, aggs = [], [], []
        for it in range(4):
            for d in dst:
                d.fill_(np.int16(np.uint16(W.POISON_BITS).view(np.int16)).item())
            pa, pb = pool.place(bpl), pool.place(bpl)
            torch.cuda.synchronize()
            pool.offload_layers(pb, 0, src_k, src_v, g.kvb, tables, sb)
            pool.wait_offloads(pb, sb)
            sb.synchronize()
            pool.synchronize()
            e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            t0 = time.perf_counter()
            e[0].record(sa)
            e[2].record(sb)
            for l in range(L):                      # interleave the two requests layer by layer, as a scheduler would
                pool.offload(pa, l, src[l][0], src[l][1], g.kvb, tables[l], sa)
                pool.retrieve(pb, l, dst[l][0], dst[l][1], g.kvb, tables[l], sb)
            pool.wait_offloads(pa, sa)
            e[1].record(sa)
            e[3].record(sb)
            torch.cuda.synchronize()
            t1 = time.perf_counter()
            if it:
                offs.append(moved / e[0].elapsed_time(e[1]) / 1e6)
                rets.append(moved / e[2].elapsed_time(e[3]) / 1e6)
                aggs.append(2 * moved / (t1 - t0) / 1e9)
            for l in range(L):
                if not torch.equal(dst[l][:, tables[l].long()], src[l][:, tables[l].long()]):
                    raise RuntimeError(f"{pname}: retrieved KV differs from the source")
            pa.release()
            pb.release()
        o, r, a = statistics.median(offs), statistics.median(rets), statistics.median(aggs)
        print(f"{pname:12s} {o:15.1f} {r:16.1f} {a:22.1f} {a / (peak_h2d + peak_d2h):14.3f}", flush=True)
    pool.destroy()


def run_blocked_io(args) -> None:
    """Blocked I/O time = time during which only KV retrieval proceeds, with no overlapping GPU computation.
    Consumer stand-in per layer = kvpool_checksum over the layer's retrieved blocks (reads K_l*P bytes through the block
    table, as decode attention does) plus an optional kvpool_spin.  Text table on stdout."""
    import torch
    from paper_2606_14779_b200 import binding as kv
    from paper_2606_14779_b200 import workloads as W

    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    spin_ns = int(args.compute_us * 1000)
    print(f"# bench.py --blocked-io --compute-us {args.compute_us}: per-layer consumer = kvpool_checksum"
          f"{' + kvpool_spin' if spin_ns else ''}; times in ms; blocked = total - consumer-alone (PAPER.md:72)")
    print("# serial = retrieve(l); consume(l); host sync, layer by layer (Fig. 2a).  pipelined = all retrieves enqueued on one stream, "
          "consume(l) on another after layer l's event (Fig. 2b).  batched = the same pipeline through ONE kvpool_retrieve_layers_signal call "
          "(the library records the per-layer events; small layers move in groups)")
    print(f"{'shape':22s} {'ctx':>7s} {'MiB':>8s} {'io_alone':>9s} {'consume':>8s} {'serial':>8s} {'blocked':>8s} {'pipelined':>9s} {'blocked':>8s} {'GB/s':>6s} {'batched':>9s} {'blocked':>8s} {'GB/s':>6s}")
    rows = []
    for cfg in (6, 3, 4):
        for ctx in (1024, 4096, 16384, 32768, 65536, 131072):
            wl = W.make_workload(cfg, scale=ctx / 131072)
            g, L = wl.geom, wl.geom.n_layers
            bw = list(wl.default_weights())
            share = np.array(bw) / np.sum(bw)
            moved = wl.moved_bytes()
            caps = [int(moved * sh * 1.25) + (L + 4) * (g.payload + 4096) for sh in share]
            pool = kv.KvPool(bw, caps, n_layers=L, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim)
            bpl = wl.blocks_per_layer(0)
            pl = pool.place(bpl)
            elems = g.kvb // 2
            src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
            dst = [W.poison_torch((2, wl.nphys, elems), dev) for l in range(L)]
            tables = [torch.from_numpy(np.ascontiguousarray(wl.layer_table(0, l))).to(dev) for l in range(L)]
            sa, sb = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
            sums = torch.zeros((4, L), dtype=torch.int64, device=dev)
            ready = [torch.cuda.Event() for _ in range(L)]
            dst_k, dst_v = [d[0] for d in dst], [d[1] for d in dst]
            torch.cuda.synchronize()        # inputs were generated on the default stream; sa / sb do not wait for it
            for l in range(L):
                pool.offload(pl, l, src[l][0], src[l][1], g.kvb, tables[l], sa)
                pool.checksum(src[l][0], src[l][1], g.kvb, tables[l], int(bpl[l]), sums[0, l:l + 1], sa)
            pool.wait_offloads(pl, sa)
            sa.synchronize()

            def consume(l, row, stream):
                pool.checksum(dst[l][0], dst[l][1], g.kvb, tables[l], int(bpl[l]), sums[row, l:l + 1], stream)
                if spin_ns:
                    pool.spin(spin_ns, stream)

            def wall(fn, reps=3):
                ts = []
                for _ in range(reps):
                    torch.cuda.synchronize()
                    pool.synchronize()
                    t0 = time.perf_counter()
                    fn()
                    torch.cuda.synchronize()
                    ts.append(1e3 * (time.perf_counter() - t0))
                return statistics.median(ts)

            def io_alone():
                for l in range(L):
                    pool.retrieve(pl, l, dst[l][0], dst[l][1], g.kvb, tables[l], sa)

            def consume_alone():
                sums[1].zero_()
                for l in range(L):
                    consume(l, 1, sb)

            def serial():
                sums[1].zero_()
                for l in range(L):
                    pool.retrieve(pl, l, dst[l][0], dst[l][1], g.kvb, tables[l], sa)
                    consume(l, 1, sa)
                    sa.synchronize()

            def pipelined():
                sums[2].zero_()
                for l in range(L):
                    pool.retrieve(pl, l, dst[l][0], dst[l][1], g.kvb, tables[l], sa)
                    e = torch.cuda.Event()
                    e.record(sa)
                    sb.wait_event(e)
                    consume(l, 2, sb)

            def pipelined_batched():        # ONE host call for the request; small layers travel in groups and become ready together
                sums[3].zero_()
                pool.retrieve_layers_signal(pl, 0, dst_k, dst_v, g.kvb, tables, ready, sa)
                for l in range(L):
                    sb.wait_event(ready[l])
                    consume(l, 3, sb)

            t_io, t_c = wall(io_alone), wall(consume_alone)
            t_ser, t_pipe, t_pb = wall(serial), wall(pipelined), wall(pipelined_batched)
            torch.cuda.synchronize()
            ok = bool(torch.equal(sums[0], sums[1]) and torch.equal(sums[0], sums[2]) and torch.equal(sums[0], sums[3]))
            if not ok:
                raise RuntimeError(f"checksum of retrieved KV differs from the source (cfg {cfg}, ctx {ctx})")
            row = {"shape": wl.name.split("@")[0], "ctx": ctx, "mib": moved / 2**20, "io_alone_ms": t_io, "consume_ms": t_c, "serial_ms": t_ser,
                   "serial_blocked_ms": t_ser - t_c, "pipelined_ms": t_pipe, "pipelined_blocked_ms": t_pipe - t_c, "pipelined_gbps": moved / t_pipe / 1e6,
                   "pipelined_batched_ms": t_pb, "pipelined_batched_blocked_ms": t_pb - t_c, "pipelined_batched_gbps": moved / t_pb / 1e6}
            rows.append(row)
            print(f"{row['shape']:22s} {ctx:7d} {row['mib']:8.0f} {t_io:9.3f} {t_c:8.3f} {t_ser:8.3f} {t_ser - t_c:8.3f} {t_pipe:9.3f} {t_pipe - t_c:8.3f} "
                  f"{row['pipelined_gbps']:6.2f} {t_pb:9.3f} {t_pb - t_c:8.3f} {row['pipelined_batched_gbps']:6.2f}", flush=True)
            pl.release()
            pool.destroy()
            del src, dst
            torch.cuda.empty_cache()
    if args.detail:
        with open(args.detail, "w") as f:
            json.dump(rows, f, indent=1)


def main():
    args = parse_args()
    if args.impl == "reference":
        print(json.dumps(run_reference(args)), flush=True)
        return
    if args.sweep:
        run_sweep(args)
        return
    if args.blocked_io:
        run_blocked_io(args)
        return
    if args.variants:
        run_variants(args)
        return
    if args.mixed_pool:
        run_mixed_pool(args)
        return
    if args.duplex:
        run_duplex(args)
        return
    out = run_kvpool(args)
    if out is None:
        return
    if not args.no_cpu_baseline and out["n_gpus"] == 1:
        out["cpu_baseline"] = cpu_baseline(args.config)
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
