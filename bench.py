#!/usr/bin/env python
"""bench.py -- Gbonds/s labeled on B200 (BASELINE.json metric), one JSON line on stdout.

A "step" is one pass of the whole hot path -- steps (i)-(iv) of PAPER.md:113 through the public C-ABI call
ccl_label_bits (ccl_label for the uint8 config 1) -- over one batch of synthetic input: the configured occupancy
sweep of the workload, one call per p.  Default workload: BASELINE.json config 5 (random 4-regular graph, 2^26
sites, 2^27 bonds, p in {0.25, 1/3, 0.45}), the configuration north_star's target is quoted on.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg1..cfg5] [--impl ours|reference]

N > 1 (under torchrun): independent replicas, one realization per rank, no data-path collective ("replicas only",
DESIGN.md section "Multi-GPU"); the value is all ranks' bonds over the slowest rank's time.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

PC_TR = 0.3473
WORKLOADS = {
    # name: (family, size parameter, z, p sweep, mask kind, BASELINE.json config number)
    "cfg1": ("honeycomb", 64, 0, [0.6527], "u8", 1),
    "cfg2": ("triangular", 4096, 0, [0.3473], "bits", 2),
    "cfg3": ("honeycomb", 4096, 0, [0.60, 0.6527, 0.70], "bits", 3),
    "cfg4": ("regular", 1 << 24, 3, [0.5], "bits", 4),
    "cfg5": ("regular", 1 << 26, 4, [0.25, 1.0 / 3.0, 0.45], "bits", 5),
    # SURVEY.md 8(f) rows, not BASELINE.json configs: the paper's own Bethe workload (Cayley tree z = 3,
    # N = 3*2^22 - 2, p = 0.5/1/1.5 p_c, standard and random numbering) and config 1 as a batch of realizations
    "cayley_std": ("cayley", 22, 0, [0.25, 0.5, 0.75], "bits", 6),
    "cayley_rand": ("cayley", 22, 1, [0.25, 0.5, 0.75], "bits", 7),
    "cfg1_batch": ("honeycomb_batch", 64, 4096, [0.6527], "bits", 1),
    # config 2 through the paper's own interface (dense NN list z_max x N, ccl_label_nn), for comparison with the bond list
    "cfg2_nn": ("triangular_nn", 4096, 0, [0.3473], "bits", 2),
}
METRIC = "Gbonds/s labeled (1 B200) and achieved HBM GB/s fraction of roofline"
SEED_BASE = 0x1603083570000000          # DESIGN.md input recipe: seed = SEED_BASE + config number
CPU_BUDGET_S = 150.0                    # reference arm: labeling time it may spend (steps are cut to fit, never the graph)


def describe(name):
    fam, size, z, ps, kind, cfg = WORKLOADS[name]
    if fam == "regular":
        n, m = size, size * z // 2
        text = "%s random %d-regular N=%d M=%d" % ("cfg%d" % cfg if cfg < 9 else "custom", z, size, m)
    elif fam == "cayley":
        n = 3 * (1 << size) - 2
        m = n - 1
        text = "Cayley tree z=3 g=%d (%s numbering) N=%d M=%d" % (size, "random" if z else "standard", n, m)
    elif fam == "honeycomb_batch":
        n, m = 2 * size * size, 3 * size * size
        text = "cfg1 honeycomb L=%d periodic N=%d M=%d x %d realizations per call (ccl_label_batch)" % (size, n, m, z)
    elif fam == "triangular_nn":
        n, m = size * size, 3 * size * size
        text = "cfg2 triangular L=%d periodic N=%d M=%d as a dense NN list (z_max x N int32, ccl_label_nn)" % (size, n, m)
    else:
        n = (2 if fam == "honeycomb" else 1) * size * size
        m = 3 * size * size
        text = "%s %s L=%d periodic N=%d M=%d" % ("cfg%d" % cfg if cfg < 9 else "custom", fam, size, n, m)
    return n, m, text + " p=" + ",".join("%.4g" % p for p in ps) + " mask=" + kind


def min_bytes(n, m, kind):
    """B_min = 8 M (src, dst) + occupancy (M/8 packed, M as uint8) + 12 N (label init write + final
    read + final write)."""
    occ = m if kind == "u8" else 4 * ((m + 31) // 32)
    return 8 * m + occ + 12 * n


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region (B200_PROFILING.md recipe), sampled through NVML from a
    thread every ~2 ms (nvidia-smi -lms needs longer to start than a whole timed region lasts here)."""
    REASONS = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index):
        self.index = index
        self.samples, self.reasons, self.smax = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        self._h = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            visible = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = int(visible.split(",")[self.index]) if visible and visible.split(",")[self.index].isdigit() else self.index
            self._h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._h = None
            return

        def run():
            import pynvml
            while not self._stop.is_set():
                try:
                    self.samples.append(float(pynvml.nvmlDeviceGetClockInfo(self._h, pynvml.NVML_CLOCK_SM)))
                    r = pynvml.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                    for name, bit in self.REASONS.items():
                        if r & bit:
                            self.reasons.add(name)
                except Exception:
                    pass
                time.sleep(0.002)
        self._thread = threading.Thread(target=run, daemon=True)
        self._thread.start()

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": self.smax, "reasons": [], "samples": 0, "how": "NVML, 2 ms period"}
        if self._thread is None:
            return out
        self._stop.set()
        self._thread.join(timeout=2)
        sm = sorted(self.samples)
        if sm:
            out.update(sm_mhz=sm[len(sm) // 2], samples=len(sm))
        out["reasons"] = sorted(self.reasons)
        return out


def oracle_inputs(name, realization=0):
    """The configured workload from the oracle's own CPU generators (untimed): (n, src, dst, [(mask, bits) per p], text)."""
    import numpy as np
    from oracle import oracle
    fam, size, z, ps, kind, cfg = WORKLOADS[name]
    seed = SEED_BASE + cfg
    if fam == "regular":
        n = size
        src, dst, _ = oracle.gen_regular(n, z, seed)
        text = "random %d-regular graph, N=2^%d sites, M=%d bonds" % (z, n.bit_length() - 1, src.size)
    elif fam == "cayley":
        n = 3 * (1 << size) - 2
        perm = np.random.default_rng(seed & 0x7FFFFFFF).permutation(n).astype(np.int32) if z else None
        n, src, dst = oracle.gen_cayley3(size, perm)
        text = "Cayley tree z=3 g=%d (%s numbering), N=%d sites, M=%d bonds" % (size, "random" if z else "standard", n, src.size)
    else:
        src, dst = (oracle.gen_honeycomb if fam.startswith("honeycomb") else oracle.gen_triangular)(size)
        n = (2 if fam.startswith("honeycomb") else 1) * size * size
        text = "%s L=%d, N=%d sites, M=%d bonds" % (fam.split("_")[0], size, n, src.size)
    reps = 64 if fam == "honeycomb_batch" else 1           # the batch workload: a bounded number of realizations per p
    masks = [oracle.gen_occupancy(src.size, p, seed, realization * reps + r) for p in ps for r in range(reps)]
    if reps > 1:
        text += " x %d realizations" % reps
    return n, src, dst, masks, text


def time_oracle(name, n, src, dst, masks, steps, warmup, budget_s=None):
    """The oracle as it stands, one thread, on the configured graph: one step = one labeling per mask of the sweep.  The
    number of steps (never the graph) is cut so that the timed labelings fit budget_s.  Returns (Gbonds/s, s per step,
    steps, warmup)."""
    from oracle import oracle
    kind = WORKLOADS[name][4]

    def sweep():
        t0 = time.perf_counter()
        for mask, bits in masks:
            if kind == "u8":
                oracle.label(n, src, dst, mask)
            else:
                oracle.label_bits(n, src, dst, bits)
        return time.perf_counter() - t0
    first = sweep()
    times = []
    if budget_s is not None:
        steps = max(1, min(steps, int(budget_s / max(first, 1e-9))))
        if first * (steps + 1) > budget_s + first:       # a sweep that takes tens of seconds is its own warm-up
            warmup = 0
    if warmup == 0:
        times.append(first)
    else:
        for _ in range(warmup - 1):
            sweep()
    while len(times) < steps:
        times.append(sweep())
    per_step = sum(times) / len(times)
    return len(masks) * src.size / per_step / 1e9, per_step, len(times), warmup


def replica_plan(rank, cfg):
    """Replicas only: every rank labels its own realization of the same workload."""
    return {"seed": SEED_BASE + cfg, "realization": rank}


def max_over_ranks(value, world, device="cpu"):
    """MAX over ranks of a host scalar (device timing): one all-reduce of the timing scalar, nothing on the data path."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world, calls_per_step, n_bonds, ms_per_step):
    """Whole-job Gbonds/s: every rank processes calls_per_step * n_bonds bonds per step, in the slowest rank's time."""
    return world * calls_per_step * n_bonds / (ms_per_step * 1e-3) / 1e9


def run_reference(args):
    """--impl reference: the oracle timed on the host cores (this tier has no other reference implementation), on the
    configured workload itself, generated by the oracle's own CPU generators."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n, m, text = describe(args.workload)
    ps = WORKLOADS[args.workload][3]
    no, src, dst, masks, what = oracle_inputs(args.workload)
    value, per_step, steps, warmup = time_oracle(args.workload, no, src, dst, masks, max(1, args.steps), max(0, min(args.warmup, 1)),
                                                 CPU_BUDGET_S)
    sample = what + ", p sweep " + ",".join("%.4g" % p for p in ps) + ", the configured graph and seeds; labeling time only, 1 thread"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "Gbonds/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": per_step * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": text, "calls_per_step": len(masks), "api": "oracle_label_bits (oracle/ccl_oracle.c)",
                   "steps_note": "steps cut to fit %.0f s of CPU labeling; the graph is never reduced" % CPU_BUDGET_S},
        "cpu_baseline": {"value": value, "unit": "Gbonds/s", "cores": 1, "kind": "oracle", "sample": sample,
                         "host_cores_available": os.cpu_count()},
        "e2e": {"value": value, "unit": "Gbonds/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


class Workload:
    """A workload resident in HBM: bond list, one occupancy mask per p, a label buffer; generated on the device by the
    library's own seeded generators (bit-identical to the oracle's: tests/test_gpu_generators_stats.py)."""

    def __init__(self, ccl, torch, name, rank):
        self.ccl, self.torch, self.name = ccl, torch, name
        self.fam, self.size, self.z, self.ps, self.kind, self.cfg = WORKLOADS[name]
        self.n, self.m, self.text = describe(name)
        fam, size, z, n, m = self.fam, self.size, self.z, self.n, self.m
        seed = SEED_BASE + self.cfg
        self.batch = z if fam == "honeycomb_batch" else 1            # realizations labeled per call
        if fam == "regular":
            self.src, self.dst = ccl.gen_regular(n, z, seed)
        elif fam == "cayley":
            perm = None
            if z:                                               # "random" numbering: a seeded permutation
                gen = torch.Generator(device="cuda")
                gen.manual_seed(seed & 0x7FFFFFFF)
                perm = torch.randperm(n, device="cuda", generator=gen).to(torch.int32)
            _, self.src, self.dst = ccl.gen_cayley3(size, perm)
        elif fam.startswith("honeycomb"):
            self.src, self.dst = ccl.gen_honeycomb(size)
        else:
            self.src, self.dst = ccl.gen_triangular(size)
        self.masks = []
        plan = replica_plan(rank, self.cfg)
        for p in self.ps:                     # replicas differ by realization = rank
            if self.batch > 1:
                words = (m + 31) // 32
                bits = torch.empty((self.batch, words), dtype=torch.int32, device="cuda")
                for r in range(self.batch):
                    bits[r] = ccl.gen_occupancy(m, p, plan["seed"], plan["realization"] * self.batch + r, want_mask=False)[1]
                self.masks.append(bits)
                continue
            mask, bits = ccl.gen_occupancy(m, p, plan["seed"], plan["realization"], want_mask=(self.kind == "u8"),
                                           want_bits=(self.kind != "u8"))
            self.masks.append(mask if self.kind == "u8" else bits)
        self.nn_lists = []
        if fam == "triangular_nn":          # NN list of the occupied bonds, every bond at both ends, built with torch ops (untimed)
            for bits in self.masks:
                b = torch.arange(m, device="cuda")
                on = ((bits[b >> 5] >> (b & 31)) & 1).bool()
                u, v = self.src[on].long(), self.dst[on].long()
                a, c = torch.cat([u, v]), torch.cat([v, u])
                a, order = torch.sort(a, stable=True)
                c = c[order]
                deg = torch.bincount(a, minlength=n)
                start = torch.cumsum(deg, 0) - deg
                slot = torch.arange(a.numel(), device="cuda") - start[a]
                nn = torch.full((int(deg.max().item()), n), -1, dtype=torch.int32, device="cuda")
                nn[slot, a] = c.to(torch.int32)
                self.nn_lists.append(nn)
                del b, on, u, v, a, c, order, deg, start, slot
        self.labels = torch.empty(n * self.batch, dtype=torch.int32, device="cuda")
        self.api = ("ccl_label_nn" if self.nn_lists else "ccl_label_batch" if self.batch > 1 else
                    "ccl_label" if self.kind == "u8" else "ccl_label_bits")
        self.stream_bytes = 8 * m + (m if self.kind == "u8" else 4 * ((m + 31) // 32))
        self.call_bytes = min_bytes(n, m, self.kind)
        if self.batch > 1:       # per call: the bond list once, a mask and 12 N of label traffic per realization
            self.stream_bytes = self.call_bytes = 8 * m + self.batch * (4 * ((m + 31) // 32) + 12 * n)
        if self.nn_lists:        # the NN list is read twice (steps (i) and (iii)) + 12 N of label traffic
            self.stream_bytes = self.call_bytes = 2 * 4 * self.nn_lists[0].numel() + 12 * n
        # L2 hygiene: the bond stream of cfg2-5 (0.2-1.1 GB) exceeds the 126 MB L2, so every call streams from HBM; for
        # the small cfg1 an L2-sized buffer is rewritten between timed calls.
        self.flush = None
        if self.call_bytes < 512 * 1024 * 1024:
            self.flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")

    def one_call(self, k):
        ccl, n = self.ccl, self.n
        if self.nn_lists:
            ccl.label_nn(self.nn_lists[k], labels=self.labels)
        elif self.batch > 1:
            ccl.label_batch(n, self.src, self.dst, self.masks[k], self.batch, labels=self.labels.view(self.batch, n))
        elif self.kind == "u8":
            ccl.label(n, self.src, self.dst, self.masks[k], labels=self.labels)
        else:
            ccl.label_bits(n, self.src, self.dst, self.masks[k], labels=self.labels)

    def cold_call_ms(self):
        """Device time of the FIRST call on this bond list: nothing remembered about it (the device-side probe runs and,
        where the call is eligible for the bucketed form, both forms are enqueued behind it) and the library's memory pool
        empty (the workspace comes from the driver).  The timed steps below are the warm-sweep steady state."""
        torch, ccl = self.torch, self.ccl
        torch.cuda.synchronize()
        ccl.set_option("probe_cache", 1)                # forgets the remembered bond lists
        ccl.trim_scratch(0)
        if self.flush is not None:
            self.flush.fill_(1)
        t0 = torch.cuda.Event(enable_timing=True)
        t1 = torch.cuda.Event(enable_timing=True)
        wall0 = time.perf_counter()
        t0.record()
        self.one_call(0)
        t1.record()
        torch.cuda.synchronize()
        return {"device_ms": t0.elapsed_time(t1), "host_wall_ms": (time.perf_counter() - wall0) * 1e3, "p": self.ps[0]}

    def measure(self, K, warmup, barrier, kernel_split=True):
        """W warm-up steps, then K timed steps (one call per p each), CUDA events on the launching stream.  Returns the
        per-call times and the per-step split the library records between its kernels."""
        torch, ccl, ps = self.torch, self.ccl, self.ps
        for _ in range(max(3, warmup)):
            for k in range(len(ps)):
                self.one_call(k)
        barrier()
        ncalls = K * len(ps)
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(ncalls)]
        split = kernel_split and self.batch == 1 and not self.nn_lists
        launches0 = ccl.launch_count()
        barrier()
        t_start = torch.cuda.Event(enable_timing=True)
        t_stop = torch.cuda.Event(enable_timing=True)
        t_start.record()
        c = 0
        for _ in range(K):
            for k in range(len(ps)):
                if self.flush is not None:
                    self.flush.fill_(c & 0xFF)
                e = ev[c]
                if not split:                                   # no per-step events inside the call
                    e[0].record(); e[1].record()
                    self.one_call(k)
                    e[2].record(); e[3].record()
                else:
                    ccl.set_profile_events(e[1], e[2], e[3])
                    e[0].record()
                    self.one_call(k)
                c += 1
        t_stop.record()
        barrier()
        launches = ccl.launch_count() - launches0
        ccl.set_profile_events(None, None, None)
        total_ms = t_start.elapsed_time(t_stop)
        call_ms = [e[0].elapsed_time(e[3]) for e in ev]
        if self.flush is not None:
            total_ms = sum(call_ms)                       # exclude the flush writes from the step time
        return {"total_ms": total_ms, "call_ms": call_ms, "init_ms": [e[0].elapsed_time(e[1]) for e in ev],
                "reduce_ms": [e[1].elapsed_time(e[2]) for e in ev], "flat_ms": [e[2].elapsed_time(e[3]) for e in ev],
                "launches": launches, "ncalls": ncalls}

    def per_p(self, r, peak):
        avg = lambda xs: sum(xs) / len(xs)
        out = {}
        n, m, batch = self.n, self.m, self.batch
        for k, p in enumerate(self.ps):
            sel = [i for i in range(r["ncalls"]) if i % len(self.ps) == k]
            t = avg([r["call_ms"][i] for i in sel])
            out["%.4g" % p] = {"ms": t, "init_ms": avg([r["init_ms"][i] for i in sel]),
                               "reduce_ms": avg([r["reduce_ms"][i] for i in sel]), "flatten_ms": avg([r["flat_ms"][i] for i in sel]),
                               "gbonds_per_s": m * batch / (t * 1e-3) / 1e9, "gsites_per_s": n * batch / (t * 1e-3) / 1e9,
                               "roofline_frac_measured": self.call_bytes / (t * 1e-3) / 1e9 / peak,
                               "roofline_frac_8TBs": self.call_bytes / (t * 1e-3) / 1e9 / 8000.0}
        return out


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_1603_08357_b200 as ccl      # raises if libccl.so cannot be built/loaded: no fallback

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    if args.region_shift >= 0 or args.force_mode >= 0:
        ccl.set_tuning(-1, args.region_shift, args.force_mode)
    for kv in args.option:
        k, v = kv.split("=")
        ccl.set_option(k, int(v))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    peak, peak_src = measured_peak()
    avg = lambda xs: sum(xs) / len(xs)
    w = Workload(ccl, torch, args.workload, rank)
    n, m, ps, kind, batch, fam, size = w.n, w.m, w.ps, w.kind, w.batch, w.fam, w.size
    torch.cuda.synchronize()
    torch.cuda.empty_cache()

    K = max(1, args.steps)
    cold = w.cold_call_ms()                 # before anything has warmed up: first call on this bond list
    sampler = ClockSampler(local)
    sampler.start()
    r = w.measure(K, args.warmup, barrier, kernel_split=not args.no_kernel_split)
    clocks = sampler.stop()
    total_ms = max_over_ranks(r["total_ms"], world, "cuda")
    ms_per_step = total_ms / K
    value = job_value(world, len(ps), m * batch, ms_per_step)
    call_ms, init_ms, reduce_ms, flat_ms, launches = r["call_ms"], r["init_ms"], r["reduce_ms"], r["flat_ms"], r["launches"]
    stream_bytes, call_bytes = w.stream_bytes, w.call_bytes
    ach = stream_bytes / (avg(reduce_ms) * 1e-3) / 1e9
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            traffic = json.load(f).get(args.workload, {}).get("k_reduce_dram_bytes_per_launch")
    except Exception:
        pass
    call_ach = call_bytes / (avg(call_ms) * 1e-3) / 1e9
    per_p = w.per_p(r, peak)

    # ---- end to end through the host-buffer entry point: H2D of the inputs and D2H of the labels inside the timing
    e2e = None
    if not args.no_e2e and kind != "u8" and batch == 1 and not w.nn_lists:
        hs, hd = w.src.cpu().pin_memory(), w.dst.cpu().pin_memory()
        hm = [b.cpu().pin_memory() for b in w.masks]
        hl = torch.empty(n, dtype=torch.int32).pin_memory()
        # the call a user makes for an occupancy sweep: ccl_label_sweep_host (bond list uploaded once, labels of mask k
        # travel back while mask k+1 is labeled); a single p goes through ccl_label_bits_host
        sweep = len(ps) > 1
        hls = [torch.empty(n, dtype=torch.int32).pin_memory() for _ in ps] if sweep else [hl]

        def e2e_step():
            if sweep:
                ccl.label_sweep_host(n, hs, hd, hm, hls)
            else:
                ccl.label_bits_host(n, hs, hd, hm[0], hl)
        e2e_step()                                                    # warm-up (memory pool, page tables)
        e2e_steps = max(5, min(K, 7))
        h2d = 2 * 4 * m + len(ps) * 4 * ((m + 31) // 32) if sweep else 2 * 4 * m + 4 * ((m + 31) // 32)
        d2h = len(ps) * 4 * n
        dts = []
        for _ in range(e2e_steps):                                    # every step synchronises: timed one by one
            barrier()
            t0 = time.perf_counter()
            e2e_step()
            torch.cuda.synchronize()
            dts.append(max_over_ranks(time.perf_counter() - t0, world, "cuda"))
        dt = sorted(dts)[len(dts) // 2]                               # the median step
        e2e = {"value": world * len(ps) * m / dt / 1e9, "unit": "Gbonds/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": e2e_steps, "statistic": "median step",
               "ms_per_step": {"median": dt * 1e3, "min": min(dts) * 1e3, "max": max(dts) * 1e3},
               "pcie_gbs_achieved": (h2d + d2h) / dt / 1e9,
               "api": ("ccl_label_sweep_host (pinned host src/dst once + one mask per p in, host labels per p out, synchronous)"
                       if sweep else "ccl_label_bits_host (pinned host src/dst/bits in, host labels out, synchronous)")}
        del hls
        del hs, hd, hm, hl
        ccl.trim_scratch(0)                                           # the host-buffer calls' device copies go back to the driver

    # ---- config 3 asks for "largest-cluster and wrapping statistics per p": untimed, after the timed region
    statistics = None
    if rank == 0 and fam in ("triangular", "honeycomb") and kind != "u8" and not w.nn_lists:
        statistics = {}
        wx, wy = ccl.gen_wrap_vectors(fam, size)
        for k, p in enumerate(ps):
            t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True); t2 = torch.cuda.Event(enable_timing=True)
            w.one_call(k)
            t0.record()
            st, _, _ = ccl.cluster_stats(w.labels, 0)
            t1.record()
            wrap_x, wrap_y, _ = ccl.wrap(n, w.src, w.dst, w.masks[k], wx, wy)
            t2.record()
            torch.cuda.synchronize()
            statistics["%.4g" % p] = {"n_clusters": st["n_clusters"], "largest": st["largest"], "largest_over_n": st["largest"] / n,
                                      "wrap_x": wrap_x, "wrap_y": wrap_y, "cluster_stats_ms": t0.elapsed_time(t1),
                                      "wrap_ms_incl_open_labeling": t1.elapsed_time(t2)}
        del wx, wy

    # ---- the oracle, one thread, on the very same graph and masks (downloaded: the device generators are bit-identical
    #      to the oracle's), timed in the same run on this host's cores
    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        import numpy as np
        reps = min(batch, 64)
        hsrc, hdst = w.src.cpu().numpy(), w.dst.cpu().numpy()
        if batch > 1:
            hmasks = [(None, np.ascontiguousarray(b[j].cpu().numpy().view(np.uint32))) for b in w.masks for j in range(reps)]
        elif kind == "u8":
            hmasks = [(b.cpu().numpy(), None) for b in w.masks]
        else:
            hmasks = [(None, np.ascontiguousarray(b.cpu().numpy().view(np.uint32))) for b in w.masks]
        v, per_step, steps_cpu, _ = time_oracle(args.workload, n, hsrc, hdst, hmasks, 1 if per_p and avg(call_ms) > 0.3 else 3,
                                                0 if n >= (1 << 22) else 1, 60.0)
        cpu = {"value": v, "unit": "Gbonds/s", "cores": 1, "kind": "oracle", "host_cores_available": os.cpu_count(),
               "seconds_per_step": per_step, "steps": steps_cpu,
               "sample": "the benchmarked workload itself (%s; same graph, same masks, downloaded from the device)%s; "
                         "labeling time only (oracle_label%s), 1 thread" % (
                             w.text, " limited to %d realizations per p" % reps if batch > 1 else "", "" if kind == "u8" else "_bits")}
        del hsrc, hdst, hmasks

    # ---- the other BASELINE.json configs, a few steps each, same timing (north_star: "report throughput on the five configs")
    configs = None
    if rank == 0 and args.workload == "cfg5" and not args.no_other_configs:
        configs = {}
        del w
        torch.cuda.empty_cache()
        for name in ("cfg1", "cfg2", "cfg3", "cfg4"):
            wk = Workload(ccl, torch, name, rank)
            torch.cuda.synchronize()
            cold_k = wk.cold_call_ms()
            rr = wk.measure(5, 3, lambda: torch.cuda.synchronize())
            t = avg(rr["call_ms"])
            configs[name] = {"workload": wk.text, "api": wk.api, "ms_per_call": t, "steps": 5, "warmup": 3,
                             "gbonds_per_s": wk.m / (t * 1e-3) / 1e9, "gsites_per_s": wk.n / (t * 1e-3) / 1e9,
                             "bytes_per_call": wk.call_bytes,
                             "roofline_call_frac": wk.call_bytes / (t * 1e-3) / 1e9 / peak,
                             "roofline_call_frac_8TBs": wk.call_bytes / (t * 1e-3) / 1e9 / 8000.0,
                             "gpu_launches_per_call": rr["launches"] / rr["ncalls"], "per_p": wk.per_p(rr, peak),
                             "cold_first_call": cold_k,
                             "l2": "256 MB buffer rewritten between timed calls" if wk.flush is not None else "inputs larger than L2"}
            del wk
            torch.cuda.empty_cache()

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": "Gbonds/s", "n_gpus": world, "steps": K,
            "warmup": max(3, args.warmup), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": describe(args.workload)[2], "calls_per_step": len(ps),
                       "api": "ccl_label_nn" if fam == "triangular_nn" else "ccl_label_batch" if batch > 1 else "ccl_label" if kind == "u8" else "ccl_label_bits",
                       "parallelism": "replicas x%d (one realization per GPU, no collective)" % world,
                       "l2": "inputs larger than L2 (bond stream %.0f MB per call vs 126 MB L2)" % (stream_bytes / 1e6)
                       if call_bytes >= 512 * 1024 * 1024 else "256 MB buffer rewritten between timed calls (L2 flush)",
                       "gsites_per_s": world * len(ps) * n * batch / (ms_per_step * 1e-3) / 1e9},
            "roofline": {"bound": "hbm", "kernel": "k_label_batch (steps i-iv)" if batch > 1 else "step (iii): k_reduce / k_hook + k_join, or k_scatter_tiles + k_descend x regions", "achieved": ach, "peak": peak, "unit": "GB/s",
                         "frac": ach / peak, "traffic": traffic, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": stream_bytes, "avg_launch_ms": avg(reduce_ms),
                         "avg_step_iii_ms": avg(reduce_ms),
                         "avg_launch_ms_is": "the event-timed duration of step (iii) of one call, which on the bucketed form is "
                                             "a chain of launches (k_scatter_tiles + one k_descend per region), not one launch; "
                                             "the largest single kernel is k_descend x regions (profiles/r2_ncu_cfg5.md: 590 of "
                                             "1224 us per call at p = 0.25)",
                         "traffic_is": "ncu dram bytes of step (iii) of ONE call at the p named in profiles/traffic.json "
                                       "(cfg5: p = 0.25 only), while achieved averages the whole p sweep",
                         "share_of_call": avg(reduce_ms) / avg(call_ms)},
            "roofline_call": {"bound": "hbm", "what": "whole ccl_label call, B_min = 8M + mask + 12N (SURVEY 8(d))",
                              "achieved": call_ach, "peak": peak, "unit": "GB/s", "frac": call_ach / peak,
                              "frac_of_8TBs_nominal": call_ach / 8000.0, "bytes_per_call": call_bytes,
                              "avg_call_ms": avg(call_ms)},
            "roofline_kernels": None if (batch > 1 or fam == "triangular_nn") else {
                "step (i) where it is a pass of its own": {"algorithmic_bytes": 4 * n, "avg_ms": avg(init_ms)},
                "step (iii)": {"algorithmic_bytes": stream_bytes, "avg_ms": avg(reduce_ms), "frac": ach / peak},
                "k_flatten (step iv)": {"algorithmic_bytes": 8 * n, "avg_ms": avg(flat_ms),
                                        "frac": 8 * n / (avg(flat_ms) * 1e-3) / 1e9 / peak}},
            "per_p": per_p, "kernel_ms": {"k_init": avg(init_ms), "k_reduce": avg(reduce_ms), "k_flatten": avg(flat_ms)},
            "configs": configs, "cold_first_call": cold,
            "timed_state": "warm sweep: the probe's answer for the bond list is remembered and the memory pool is reserved "
                           "(>= 3 warm-up sweeps on the same src/dst); cold_first_call is the first call without either",
            "statistics": statistics, "clocks": clocks, "e2e": e2e, "cpu_baseline": cpu, "gpu_launches": launches,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg5", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--family", choices=["triangular", "honeycomb", "regular", "cayley"],
                    help="a workload outside the table: --family with --size (L, or sites for regular, or generations for "
                         "cayley), --z (degree; cayley: 1 = random numbering) and --p (comma-separated); used for the "
                         "paper's own sizes (PAPER.md:171-173, 193)")
    ap.add_argument("--size", type=int, default=0)
    ap.add_argument("--z", type=int, default=0)
    ap.add_argument("--p", default="")
    ap.add_argument("--region-shift", type=int, default=-1, help="experiment: log2 sites per region of the bucketed form")
    ap.add_argument("--force-mode", type=int, default=-1, help="experiment: -1 probe, 0 direct, 1 bucketed")
    ap.add_argument("--option", action="append", default=[], help="experiment: name=value for ccl_set_option")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-kernel-split", action="store_true",
                    help="do not record events between the kernels of a call (an event record between two kernels keeps them "
                         "from overlapping by programmatic dependent launch)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="cfg5 only: do not also measure cfg1-cfg4 afterwards")
    args = ap.parse_args()
    if args.family:
        ps = [float(t) for t in args.p.split(",") if t]
        if not ps or args.size <= 0:
            ap.error("--family needs --size and --p")
        WORKLOADS["custom"] = (args.family, args.size, args.z, ps, "bits", 9)
        args.workload = "custom"
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
