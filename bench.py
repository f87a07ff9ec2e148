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
CPU_SAMPLE_LOG2_SITES = 22              # cpu_baseline / reference arm: same family at 2^22 sites (bounded sample)


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


def cpu_oracle_sample(name, steps, warmup):
    """The oracle as it stands, single thread, on a bounded sample of the workload; returns (Gbonds/s, seconds per
    step, description).  Lattice workloads are sampled at L = 1024, the regular graphs at 2^22 sites."""
    import numpy as np  # noqa: F401
    from oracle import oracle
    fam, size, z, ps, kind, cfg = WORKLOADS[name]
    seed = SEED_BASE + cfg
    if fam == "regular":
        n = min(size, 1 << CPU_SAMPLE_LOG2_SITES)
        src, dst, _ = oracle.gen_regular(n, z, seed)
        sample = "random %d-regular graph, N=2^%d sites, M=%d bonds" % (z, n.bit_length() - 1, src.size)
    elif fam == "cayley":
        g = min(size, 20)
        n = 3 * (1 << g) - 2
        perm = np.random.default_rng(seed & 0x7FFFFFFF).permutation(n).astype(np.int32) if z else None
        n, src, dst = oracle.gen_cayley3(g, perm)
        sample = "Cayley tree z=3 g=%d (%s numbering), N=%d sites, M=%d bonds" % (g, "random" if z else "standard", n, src.size)
    else:
        L = min(size, 1024)
        src, dst = (oracle.gen_honeycomb if fam.startswith("honeycomb") else oracle.gen_triangular)(L)
        n = (2 if fam.startswith("honeycomb") else 1) * L * L
        sample = "%s L=%d, N=%d sites, M=%d bonds (bond-list oracle)" % (fam, L, n, src.size)
    reps = 256 if fam == "honeycomb_batch" else 1           # a bounded sample of the batch: 256 realizations per p
    masks = [oracle.gen_occupancy(src.size, p, seed, r) for p in ps for r in range(reps)]
    if reps > 1:
        sample += " x %d realizations" % reps
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        for mask, bits in masks:
            if kind == "u8":
                oracle.label(n, src, dst, mask)
            else:
                oracle.label_bits(n, src, dst, bits)
        if it >= warmup:
            times.append(time.perf_counter() - t0)
    per_step = sum(times) / len(times)
    sample += ", p sweep " + ",".join("%.4g" % p for p in ps) + ", same seeds; labeling time only (oracle_label%s)" % (
        "" if kind == "u8" else "_bits")
    return len(masks) * src.size / per_step / 1e9, per_step, sample


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
    """--impl reference: the oracle timed on the host cores (this tier has no other reference implementation)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n, m, text = describe(args.workload)
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    # keep the whole run within a few minutes: a 2^22-site sweep costs about 2 s per step
    steps_eff, warmup_eff = min(steps, 20), min(warmup, 3)
    value, per_step, sample = cpu_oracle_sample(args.workload, steps_eff, warmup_eff)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "Gbonds/s", "n_gpus": args.gpus,
        "steps": steps_eff, "warmup": warmup_eff, "ms_per_step": per_step * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": {"workload": text, "sample": sample},
        "cpu_baseline": {"value": value, "unit": "Gbonds/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "Gbonds/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


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

    fam, size, z, ps, kind, cfg = WORKLOADS[args.workload]
    n, m, text = describe(args.workload)
    seed = SEED_BASE + cfg
    if args.region_shift >= 0 or args.force_mode >= 0:
        ccl.set_tuning(-1, args.region_shift, args.force_mode)
    for kv in args.option:
        k, v = kv.split("=")
        ccl.set_option(k, int(v))
    # ---- synthetic inputs, generated on the device by the library's own seeded generators (untimed)
    batch = z if fam == "honeycomb_batch" else 1            # realizations labeled per call
    if fam == "regular":
        src, dst = ccl.gen_regular(n, z, seed)
    elif fam == "cayley":
        perm = None
        if z:                                               # "random" numbering: a seeded permutation
            gen = torch.Generator(device="cuda")
            gen.manual_seed(seed & 0x7FFFFFFF)
            perm = torch.randperm(n, device="cuda", generator=gen).to(torch.int32)
        _, src, dst = ccl.gen_cayley3(size, perm)
    elif fam.startswith("honeycomb"):
        src, dst = ccl.gen_honeycomb(size)
    else:
        src, dst = ccl.gen_triangular(size)
    masks = []
    plan = replica_plan(rank, cfg)
    for p in ps:                      # replicas differ by realization = rank
        if batch > 1:
            words = (m + 31) // 32
            bits = torch.empty((batch, words), dtype=torch.int32, device="cuda")
            for r in range(batch):
                bits[r] = ccl.gen_occupancy(m, p, plan["seed"], plan["realization"] * batch + r, want_mask=False)[1]
            masks.append(bits)
            continue
        mask, bits = ccl.gen_occupancy(m, p, plan["seed"], plan["realization"], want_mask=(kind == "u8"),
                                       want_bits=(kind != "u8"))
        masks.append(mask if kind == "u8" else bits)
    nn_lists = []
    if fam == "triangular_nn":          # NN list of the occupied bonds, every bond at both ends, built with torch ops (untimed)
        for bits in masks:
            b = torch.arange(m, device="cuda")
            on = ((bits[b >> 5] >> (b & 31)) & 1).bool()
            u, v = src[on].long(), dst[on].long()
            a, c = torch.cat([u, v]), torch.cat([v, u])
            a, order = torch.sort(a, stable=True)
            c = c[order]
            deg = torch.bincount(a, minlength=n)
            start = torch.cumsum(deg, 0) - deg
            slot = torch.arange(a.numel(), device="cuda") - start[a]
            nn = torch.full((int(deg.max().item()), n), -1, dtype=torch.int32, device="cuda")
            nn[slot, a] = c.to(torch.int32)
            nn_lists.append(nn)
            del b, on, u, v, a, c, order, deg, start, slot
    labels = torch.empty(n * batch, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    torch.cuda.empty_cache()

    def one_call(k):
        if nn_lists:
            ccl.label_nn(nn_lists[k], labels=labels)
        elif batch > 1:
            ccl.label_batch(n, src, dst, masks[k], batch, labels=labels.view(batch, n))
        elif kind == "u8":
            ccl.label(n, src, dst, masks[k], labels=labels)
        else:
            ccl.label_bits(n, src, dst, masks[k], labels=labels)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # L2 hygiene: the bond stream of cfg2-5 (0.2-1.1 GB) exceeds the 126 MB L2, so every call streams from HBM; for
    # the small cfg1 an L2-sized buffer is rewritten between timed calls.
    flush = None
    if min_bytes(n, m, kind) < 512 * 1024 * 1024:
        flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")

    for _ in range(max(3, args.warmup)):
        for k in range(len(ps)):
            one_call(k)
    barrier()

    K = max(1, args.steps)
    ncalls = K * len(ps)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(ncalls)]
    sampler = ClockSampler(local)
    sampler.start()
    launches0 = ccl.launch_count()
    barrier()
    t_start = torch.cuda.Event(enable_timing=True)
    t_stop = torch.cuda.Event(enable_timing=True)
    flush_ms = 0.0
    t_start.record()
    c = 0
    for _ in range(K):
        for k in range(len(ps)):
            if flush is not None:
                flush.fill_(c & 0xFF)
            e = ev[c]
            if batch > 1 or nn_lists or args.no_kernel_split:   # no per-step events inside the call
                e[0].record(); e[1].record()
                one_call(k)
                e[2].record(); e[3].record()
            else:
                ccl.set_profile_events(e[1], e[2], e[3])
                e[0].record()
                one_call(k)
            c += 1
    t_stop.record()
    barrier()
    launches = ccl.launch_count() - launches0
    clocks = sampler.stop()
    ccl.set_profile_events(None, None, None)
    total_ms = t_start.elapsed_time(t_stop)
    call_ms = [e[0].elapsed_time(e[3]) for e in ev]
    init_ms = [e[0].elapsed_time(e[1]) for e in ev]
    reduce_ms = [e[1].elapsed_time(e[2]) for e in ev]
    flat_ms = [e[2].elapsed_time(e[3]) for e in ev]
    if flush is not None:
        total_ms = sum(call_ms)                       # exclude the flush writes from the step time
    total_ms = max_over_ranks(total_ms, world, "cuda")
    ms_per_step = total_ms / K
    value = job_value(world, len(ps), m * batch, ms_per_step)

    peak, peak_src = measured_peak()
    avg = lambda xs: sum(xs) / len(xs)
    stream_bytes = 8 * m + (m if kind == "u8" else 4 * ((m + 31) // 32))
    call_bytes = min_bytes(n, m, kind)
    if batch > 1:            # per call: the bond list once, a mask and 12 N of label traffic per realization
        stream_bytes = call_bytes = 8 * m + batch * (4 * ((m + 31) // 32) + 12 * n)
    if nn_lists:             # the NN list is read twice (steps (i) and (iii)) + 12 N of label traffic
        stream_bytes = call_bytes = 2 * 4 * nn_lists[0].numel() + 12 * n
    ach = stream_bytes / (avg(reduce_ms) * 1e-3) / 1e9
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            traffic = json.load(f).get(args.workload, {}).get("k_reduce_dram_bytes_per_launch")
    except Exception:
        pass
    call_ach = call_bytes / (avg(call_ms) * 1e-3) / 1e9
    per_p = {}
    for k, p in enumerate(ps):
        sel = [i for i in range(ncalls) if i % len(ps) == k]
        t = avg([call_ms[i] for i in sel])
        per_p["%.4g" % p] = {"ms": t, "init_ms": avg([init_ms[i] for i in sel]),
                             "reduce_ms": avg([reduce_ms[i] for i in sel]), "flatten_ms": avg([flat_ms[i] for i in sel]),
                             "gbonds_per_s": m * batch / (t * 1e-3) / 1e9, "gsites_per_s": n * batch / (t * 1e-3) / 1e9,
                             "roofline_frac_measured": call_bytes / (t * 1e-3) / 1e9 / peak,
                             "roofline_frac_8TBs": call_bytes / (t * 1e-3) / 1e9 / 8000.0}

    # ---- end to end through the host-buffer entry point: H2D of the inputs and D2H of the labels inside the timing
    e2e = None
    if not args.no_e2e and kind != "u8" and batch == 1 and not nn_lists:
        hs, hd = src.cpu().pin_memory(), dst.cpu().pin_memory()
        hm = [b.cpu().pin_memory() for b in masks]
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
        e2e_steps = max(1, min(K, 3))
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dt, world, "cuda")
        h2d = 2 * 4 * m + len(ps) * 4 * ((m + 31) // 32) if sweep else 2 * 4 * m + 4 * ((m + 31) // 32)
        d2h = len(ps) * 4 * n
        e2e = {"value": world * len(ps) * m * e2e_steps / dt / 1e9, "unit": "Gbonds/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": e2e_steps,
               "api": ("ccl_label_sweep_host (pinned host src/dst once + one mask per p in, host labels per p out, synchronous)"
                       if sweep else "ccl_label_bits_host (pinned host src/dst/bits in, host labels out, synchronous)")}
        del hls
        del hs, hd, hm, hl

    # ---- config 3 asks for "largest-cluster and wrapping statistics per p": untimed, after the timed region
    statistics = None
    if rank == 0 and fam in ("triangular", "honeycomb") and kind != "u8" and not nn_lists:
        statistics = {}
        wx, wy = ccl.gen_wrap_vectors(fam, size)
        for k, p in enumerate(ps):
            t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True); t2 = torch.cuda.Event(enable_timing=True)
            one_call(k)
            t0.record()
            st, _, _ = ccl.cluster_stats(labels, 0)
            t1.record()
            wrap_x, wrap_y, _ = ccl.wrap(n, src, dst, masks[k], wx, wy)
            t2.record()
            torch.cuda.synchronize()
            statistics["%.4g" % p] = {"n_clusters": st["n_clusters"], "largest": st["largest"], "largest_over_n": st["largest"] / n,
                                      "wrap_x": wrap_x, "wrap_y": wrap_y, "cluster_stats_ms": t0.elapsed_time(t1),
                                      "wrap_ms_incl_open_labeling": t1.elapsed_time(t2)}
        del wx, wy

    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        v, per_step, sample = cpu_oracle_sample(args.workload, 3, 1)
        cpu = {"value": v, "unit": "Gbonds/s", "cores": 1, "kind": "oracle", "sample": sample,
               "host_cores_available": os.cpu_count()}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": "Gbonds/s", "n_gpus": world, "steps": K,
            "warmup": max(3, args.warmup), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": text, "calls_per_step": len(ps), "api": "ccl_label_nn" if nn_lists else "ccl_label_batch" if batch > 1 else "ccl_label" if kind == "u8" else "ccl_label_bits",
                       "parallelism": "replicas x%d (one realization per GPU, no collective)" % world,
                       "l2": "inputs larger than L2 (bond stream %.0f MB per call vs 126 MB L2)" % (stream_bytes / 1e6)
                       if flush is None else "256 MB buffer rewritten between timed calls (L2 flush)",
                       "gsites_per_s": world * len(ps) * n * batch / (ms_per_step * 1e-3) / 1e9},
            "roofline": {"bound": "hbm", "kernel": "k_label_batch (steps i-iv)" if batch > 1 else "step (iii): k_reduce, or k_scatter + k_descend x regions", "achieved": ach, "peak": peak, "unit": "GB/s",
                         "frac": ach / peak, "traffic": traffic, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": stream_bytes, "avg_launch_ms": avg(reduce_ms),
                         "share_of_call": avg(reduce_ms) / avg(call_ms)},
            "roofline_call": {"bound": "hbm", "what": "whole ccl_label call, B_min = 8M + mask + 12N (SURVEY 8(d))",
                              "achieved": call_ach, "peak": peak, "unit": "GB/s", "frac": call_ach / peak,
                              "frac_of_8TBs_nominal": call_ach / 8000.0, "bytes_per_call": call_bytes,
                              "avg_call_ms": avg(call_ms)},
            "roofline_kernels": None if (batch > 1 or nn_lists) else {
                "k_init (step i)": {"algorithmic_bytes": 4 * n, "avg_ms": avg(init_ms),
                                    "frac": 4 * n / (avg(init_ms) * 1e-3) / 1e9 / peak},
                "step (iii)": {"algorithmic_bytes": stream_bytes, "avg_ms": avg(reduce_ms), "frac": ach / peak},
                "k_flatten (step iv)": {"algorithmic_bytes": 8 * n, "avg_ms": avg(flat_ms),
                                        "frac": 8 * n / (avg(flat_ms) * 1e-3) / 1e9 / peak}},
            "per_p": per_p, "kernel_ms": {"k_init": avg(init_ms), "k_reduce": avg(reduce_ms), "k_flatten": avg(flat_ms)},
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
