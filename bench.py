#!/usr/bin/env python
"""bench.py -- one JSON line (< 4 KB) for the SPH offload hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload default|config1|config2|config3|config4|link|layouts|...]

The default line is on BASELINE.json:configs[4], the largest single-GPU configuration and the B200 counterpart of the paper's
whole offload cycle: 2^26 particles, per step pack -> density -> unpack -> ghost -> pack -> force -> unpack in
bundles of 4,096 tasks over two streams.  `value` = particles/s through that step with the store resident in HBM (whole job: all
ranks' particles / max-over-ranks time); `e2e` = the same step with the store in pinned HOST memory through the C-ABI calls, every
host<->device copy inside the timed region; `roofline` = the dominant kernel (the force loop) against the FP32 peak; `kernels` =
name -> fraction of its roofline for the stages of this step and (N = 1) for configs[2]'s pack / force / unpack in both layouts and
configs[3]'s streamed pack / unpack against the host link.  Everything else -- per-stage tables, the other configurations -- is
written to gpurun_out/bench_side.json, never to stdout.  (--workload X runs one configuration and prints its own line.)
--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same configs[4] input.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particles/s pack+unpack and pair-interactions/s; % of HBM / host-link roofline"
CONFIG1_NAME = "configs[1]: 262144 particles, 64^3 glass-like lattice, 16^3 cells, density loop then force loop"
SHARDING = "one independent box per rank, no collective"
N_SM, LANES_PER_SM = 148, 128
# algorithmic FP32 work of the loops: 8 flop per ordered candidate pair (3 sub, 1 mul,
# 2 fma, 1 compare) + per neighbour hit 25 flop (density) / 60 flop (force)
FLOP_CAND, FLOP_HIT_DENSITY, FLOP_HIT_FORCE, FLOP_HIT_GRADIENT = 8.0, 25.0, 60.0, 45.0
NGB_CONFIG1 = 63.04    # (32/3) pi (1.2348)^3: neighbours per particle incl. self at h = 1.2348 dx


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """SM clock / throttle-reason samples taken DURING the timed region (B200_PROFILING.md's clocks line).

    A thread polls NVML (nvidia_ml_py) every millisecond, so even a timed region of a few milliseconds is sampled;
    if NVML cannot be loaded it falls back to one `nvidia-smi -lms 100` process."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        import threading
        self.sm, self.reasons, self.max_mhz = [], set(), None
        self.p = self.f = self.thread = None
        self._stop = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            phys = int(vis.split(",")[index]) if vis and all(t.strip().isdigit() for t in vis.split(",")) else index
            h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            bits = {"hw_slowdown": pynvml.nvmlClocksThrottleReasonHwSlowdown, "hw_thermal_slowdown": pynvml.nvmlClocksThrottleReasonHwThermalSlowdown,
                    "sw_thermal_slowdown": pynvml.nvmlClocksThrottleReasonSwThermalSlowdown, "sw_power_cap": pynvml.nvmlClocksThrottleReasonSwPowerCap}

            def poll():
                while not self._stop.is_set():
                    try:
                        self.sm.append(float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)))
                        r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                        for name, bit in bits.items():
                            if r & bit:
                                self.reasons.add(name)
                    except Exception:
                        pass
                    time.sleep(0.001)
            self.thread = threading.Thread(target=poll, daemon=True)
            self.thread.start()
        except Exception:
            self.thread = None
            self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            try:
                self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100", "-i", str(index)],
                                          stdout=self.f, stderr=subprocess.DEVNULL)
            except OSError:
                pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        if self.thread is not None:
            self._stop.set()
            self.thread.join(timeout=2)
        elif self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.p.kill()
            self.f.flush()
            rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
            os.unlink(self.f.name)
            for r in rows:
                if len(r) < 9:
                    continue
                try:
                    self.sm.append(float(r[1]))
                    out["sm_max_mhz"] = float(r[2])
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                    if v.strip().lower() == "active":
                        self.reasons.add(name)
        if self.sm:
            out["sm_mhz"] = statistics.median(self.sm)
        out["reasons"], out["samples"] = sorted(self.reasons), len(self.sm)
        return out


def dist_setup(n_gpus):
    """one process per GPU under torchrun; returns (rank, world, device index)"""
    import torch
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    if world > 1:
        import torch.distributed as dist
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        if torch.cuda.is_available():
            torch.cuda.set_device(local)
        dist.init_process_group(backend=backend)
    return rank, world, local


def dist_barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def dist_max(value, world, device="cpu"):
    """max over ranks of a python float (timing rule: the slowest rank defines the step)"""
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def dist_sum(value, world, device="cpu"):
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# --------------------------------------------------------------------------------------------- our arm

class Workload:
    """configs[1] resident on the current device in one layout, one batch holding every task of a loop; the two-loop cycle
    (density, force) or the three-loop cycle (density, gradient, Balsara-switched force: PAPER.md:41, reading C34)."""

    def __init__(self, sph, torch, ps, cells, tasks, layout_name, loops=2):
        self.sph, self.torch = sph, torch
        self.layout_name, self.loops = layout_name, loops
        from paper_2606_23891_b200 import layouts as _layouts
        self.layout = _layouts.layout(sph, layout_name, loops=loops)
        self.n = ps.shape[0]
        self.cells = cells
        self.store = sph.sph_store_create(self.layout, self.n)
        sph.sph_store_import_aos(self.store, ps)
        sph.sph_store_set_cells(self.store, cells)
        self.batch = sph.sph_batch_create(self.store, tasks)
        self.info = sph.sph_batch_get_info(self.batch)
        self.sets = [sph.sph_attrset_canonical(k) for k in range(7 if loops == 3 else 4)]
        self.rec = [sph.sph_attrset_record_bytes(s) for s in self.sets]
        self.bufs = [torch.empty(sph.sph_batch_buffer_bytes(self.batch, s), dtype=torch.uint8, device="cuda") for s in self.sets]
        self.params = sph.sph_params(np.float32(5.0 / 3.0), 0.8, 3.0)
        # host mirrors of the substruct arrays for the end-to-end leg (pinned)
        self.host = []
        for s in range(self.layout.n_sub):
            nb = self.n * self.layout.stride[s]
            h = torch.empty(nb, dtype=torch.uint8).pin_memory()
            self.host.append(h)
        # which substructs a step reads from / writes to the host copy
        f = sph.FIELD
        sub = lambda names: {self.layout.loc[f[k]].sub for k in names}
        self.sub = sub
        ins = sub(("x", "h", "mass", "v", "u") + (("time_bin",) if loops == 3 else ()))
        outs = sub(("rho", "rho_dh", "wcount", "wcount_dh", "P", "c_s", "a", "du_dt", "v_sig") + (("div_v", "rot_v") if loops == 3 else ()))
        self.subs_in, self.subs_out = sorted(ins), sorted(outs)
        for s in range(self.layout.n_sub):
            sph.sph_store_download_sub(self.store, s, self.host[s])
        torch.cuda.synchronize()

    # the launches of a step, as (name, callable): seven (two loops) or ten (three loops)
    def launches(self, stream=None):
        stream = stream if stream is not None else self.torch.cuda.current_stream()
        sph, st, b, S, B, p = self.sph, self.store, self.batch, self.sets, self.bufs, self.params
        # "zero the outputs of the loop about to run" is fused into the unpack (SPH_UNPACK_REDUCE_ZERO: one batch holds the whole
        # loop, so every particle's sums start from 0 there) -- bit-identical to sph_store_zero + SPH_UNPACK_REDUCE
        Z = sph.SPH_UNPACK_REDUCE_ZERO
        head = [
            ("pack_density_in", lambda: sph.sph_pack(st, b, S[0], B[0], stream)),
            ("density", lambda: sph.sph_density(b, B[0], B[1], stream)),
            ("unpack_density_out", lambda: sph.sph_unpack(st, b, S[1], B[1], Z, stream)),
            ("ghost", lambda: sph.sph_ghost(st, p, stream)),
        ]
        if self.loops == 3:
            return head + [
                ("pack_gradient_in", lambda: sph.sph_pack(st, b, S[4], B[4], stream)),
                ("gradient", lambda: sph.sph_gradient(b, B[4], B[5], stream)),
                ("unpack_gradient_out", lambda: sph.sph_unpack(st, b, S[5], B[5], Z, stream)),
                ("pack_force_in", lambda: sph.sph_pack(st, b, S[6], B[6], stream)),
                ("force", lambda: sph.sph_force3(b, B[6], B[3], p, stream)),
                ("unpack_force_out", lambda: sph.sph_unpack(st, b, S[3], B[3], Z, stream)),
            ]
        return head + [
            ("pack_force_in", lambda: sph.sph_pack(st, b, S[2], B[2], stream)),
            ("force", lambda: sph.sph_force(b, B[2], B[3], p, stream)),
            ("unpack_force_out", lambda: sph.sph_unpack(st, b, S[3], B[3], Z, stream)),
        ]

    def step(self, stream=None):
        for _, fn in self.launches(stream):
            fn()

    def step_e2e(self, stream=None):
        """The step with the particle arrays in pinned HOST memory.  Uploads run on a copy stream ahead of the kernels that need
        them, downloads on a second one as soon as a substruct holds its final values, so that with split-AoS the later loops'
        inputs cross during the density loop and each loop's results during the next loop; the first pack and the last unpack
        are streamed in four slabs of cells (sph_pack_cells / sph_unpack_cells) against their copies.  A substruct that holds
        both a later loop's inputs and an earlier loop's outputs (pack-density, pack-gradient, ...) is uploaded BEFORE the
        kernel that writes those outputs runs.  The calling stream waits for the last download: its events bracket the step."""
        torch, sph = self.torch, self.sph
        main = stream if stream is not None else torch.cuda.current_stream()
        if not hasattr(self, "_e2e"):
            sub = self.sub
            d_in = sub(("x", "h", "mass"))
            later_in = sub(("v", "u") + (("time_bin",) if self.loops == 3 else ())) - d_in
            # the stages that write the store, in order, and the substructs each one writes
            writes = [("unpack_density_out", sub(("rho", "rho_dh", "wcount", "wcount_dh"))), ("ghost", sub(("P", "c_s")))]
            if self.loops == 3:
                writes.append(("unpack_gradient_out", sub(("div_v", "rot_v"))))
            writes.append(("unpack_force_out", sub(("a", "du_dt", "v_sig"))))
            last = {}
            for k, subs in writes:
                for s_ in subs:
                    last[s_] = k                      # a substruct leaves after the last stage that writes it
            written = set().union(*[subs for _, subs in writes])
            self._e2e = {"up": torch.cuda.Stream(), "down": torch.cuda.Stream(), "up1": sorted(d_in), "up2": sorted(later_in),
                         "down_after": {k: sorted(s_ for s_, kk in last.items() if kk == k) for k, _ in writes},
                         # the later loops' inputs must have landed before the first kernel that writes their substruct (else
                         # before the first kernel that reads them: the ghost reads u)
                         "up2_before": next((k for k, subs in writes if subs & later_in), None) if later_in & written else None}
            from bench_workloads import cell_slabs
            self._e2e["slabs"] = cell_slabs(self.cells, 4)
        E = self._e2e
        up, down = E["up"], E["down"]
        ev = lambda st: (lambda e: (e.record(st), e)[1])(torch.cuda.Event())
        start = ev(main)
        up.wait_event(start)
        down.wait_event(start)
        # the density inputs cross slab by slab (ranges of cells); each slab is packed as soon as it is there
        S, B, st, b = self.sets, self.bufs, self.store, self.batch
        for c0, nc, p0, npart in E["slabs"]:
            for s in E["up1"]:
                sph.sph_store_upload_range(st, s, self.host[s], p0, npart, up)
            main.wait_event(ev(up))
            sph.sph_pack_cells(st, b, S[0], B[0], c0, nc, main)
        for s in E["up2"]:
            sph.sph_store_upload_sub(self.store, s, self.host[s], up)
        e2 = ev(up)
        waited = False
        for k, fn in self.launches(main)[1:]:
            if not waited and k in (E["up2_before"], "ghost"):        # the ghost reads u
                main.wait_event(e2)
                waited = True
            if k == "unpack_force_out":
                break
            fn()
            if E["down_after"].get(k):
                down.wait_event(ev(main))
                for s in E["down_after"][k]:
                    sph.sph_store_download_sub(self.store, s, self.host[s], down)
        # the force results are reduced slab by slab; each slab's particles leave as soon as they are final
        for c0, nc, p0, npart in E["slabs"]:
            sph.sph_unpack_cells(st, b, S[3], B[3], c0, nc, sph.SPH_UNPACK_REDUCE_ZERO, main)
            down.wait_event(ev(main))
            for s in E["down_after"]["unpack_force_out"]:
                sph.sph_store_download_range(st, s, self.host[s], p0, npart, down)
        main.wait_event(ev(down))

    def capture_e2e(self):
        """step_e2e captured once as a CUDA graph (copies, kernels and the cross-stream events): a replay costs one launch on
        the host instead of ~50 calls through ctypes, which would otherwise bound a 0.9 ms step"""
        torch = self.torch
        root = torch.cuda.Stream()
        with torch.cuda.stream(root):
            self.step_e2e(root)                      # warm-up outside the capture (first-call attribute setting)
        torch.cuda.synchronize()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph, stream=root):
            self.step_e2e(root)
        return self.graph

    def e2e_bytes(self):
        return (sum(self.n * self.layout.stride[s] for s in self.subs_in), sum(self.n * self.layout.stride[s] for s in self.subs_out))

    def algorithmic(self):
        """algorithmic bytes / flop per launch: every record byte once, every touched store
        field once per particle per launch (re-reads of a cell by its 27 tasks are cache hits, not algorithmic traffic)."""
        n, inst, cand = self.n, self.info.n_instances, self.info.n_candidates
        r = self.rec
        F = self.sph.FIELD
        width = lambda f: 8 if f in (F["x"], F["id"]) else (1 if f == F["time_bin"] else 4)
        fields_in = lambda k: sum(int(e.ncomp) * width(int(e.field)) for e in list(self.sets[k].ent)[:self.sets[k].n])      # store bytes read per particle
        out = {
            "pack_density_in": {"bound": "hbm", "bytes": n * 32 + inst * r[0]},
            "unpack_density_out": {"bound": "hbm", "bytes": inst * r[1] + n * 16},       # REDUCE_ZERO: the fields are written, not read
            "unpack_force_out": {"bound": "hbm", "bytes": inst * r[3] + n * 20},
            "density": {"bound": "alu", "flop": cand * FLOP_CAND + n * NGB_CONFIG1 * FLOP_HIT_DENSITY},
            "force": {"bound": "alu", "flop": cand * FLOP_CAND + n * (NGB_CONFIG1 - 1) * FLOP_HIT_FORCE},
        }
        if self.loops == 3:
            out["pack_gradient_in"] = {"bound": "hbm", "bytes": n * fields_in(4) + inst * r[4]}
            out["unpack_gradient_out"] = {"bound": "hbm", "bytes": inst * r[5] + n * 16}
            out["pack_force_in"] = {"bound": "hbm", "bytes": n * fields_in(6) + inst * r[6]}
            out["gradient"] = {"bound": "alu", "flop": cand * FLOP_CAND + n * (NGB_CONFIG1 - 1) * FLOP_HIT_GRADIENT}
        else:
            out["pack_force_in"] = {"bound": "hbm", "bytes": n * 64 + inst * r[2]}
        return out

    def close(self):
        self.graph = None
        self.sph.sph_batch_destroy(self.batch)
        self.sph.sph_store_destroy(self.store)


def build_config1(sph, seed):
    import sph_inputs as si
    parts = si.config1(seed=seed)
    perm, cells = sph.sph_cells_build_grid(parts["x"], 16)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    hmax = np.full(cells.shape[0], ps["h"].max(), dtype=np.float32)      # constant h in configs[1]
    tasks, n_self, n_pair = sph.sph_tasks_build(cells, hmax)
    return ps, cells, tasks


def time_steps(torch, fn, steps, warmup, flush, world):
    """per-step CUDA-event times [ms]; L2 flushed (untimed) before every step; barrier + sync on both sides"""
    for _ in range(warmup):
        flush()
        fn()
    torch.cuda.synchronize()
    dist_barrier(world)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        flush()
        a.record()
        fn()
        b.record()
    torch.cuda.synchronize()
    dist_barrier(world)
    return [a.elapsed_time(b) for a, b in ev]


def same_size_copy_gbs(torch, nbytes, flush, reps=7):
    """The yardstick for one HBM-bound launch of `nbytes` algorithmic bytes: a device-to-device copy that moves the same bytes
    (half read, half written; torch's copy kernel) as ONE launch on a flushed L2, timed with CUDA events the way the kernels
    are.  The MEASURED_PEAKS figure is a 4 GiB copy; a launch of 100-400 MB pays its ramp-up and tail on a cold L2."""
    half = max(1 << 20, int(nbytes) // 2)
    a = torch.empty(half, dtype=torch.uint8, device="cuda")
    b = torch.empty(half, dtype=torch.uint8, device="cuda")
    best = None
    for _ in range(reps):
        flush()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); b.copy_(a); e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    return 2 * half / (best * 1e-3) / 1e9


def same_size_fill_gbs(torch, nbytes, flush, reps=7):
    """The write-only yardstick (a pack launch is ~94 % writes): torch's fill kernel over the same number of bytes, one launch on a
    flushed L2, timed the same way.  HBM writes run below the read + write copy figure."""
    a = torch.empty(max(1 << 20, int(nbytes)), dtype=torch.uint8, device="cuda")
    best = None
    for _ in range(reps):
        flush()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); a.fill_(3); e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    return a.numel() / (best * 1e-3) / 1e9


def run_other_workload(args):
    """configs[2..4] and the link probe (bench_workloads.py); single GPU, same JSON contract"""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    if int(os.environ.get("RANK", 0)) != 0:
        return
    import paper_2606_23891_b200 as sph
    import bench_workloads as bw
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", 0)))
    hbm_peak, sm_max_mhz, peak_src = measured_peaks()
    common = {"hbm_peak": hbm_peak, "alu_peak": N_SM * LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12, "peak_source": peak_src,
              "time_steps": lambda torch_, fn, steps, warmup, flush: time_steps(torch_, fn, steps, warmup, flush, 1), "sampler": lambda: None}
    sampler = ClockSampler(0)
    body = bw.RUNNERS[args.workload](args, sph, torch, common)
    clocks = sampler.stop()
    line = {"metric": METRIC, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "data": "synthetic", "clocks": clocks, "peak_source": peak_src}
    line.update(body)
    print(json.dumps(line))


def run_layouts(args):
    """configs[1] through every particle layout of the paper (Fig. 2's axis): pack + unpack time per layout
    in HBM, the whole step, and the end-to-end step with the store's arrays in pinned host memory"""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    if int(os.environ.get("RANK", 0)) != 0:
        return
    import paper_2606_23891_b200 as sph
    from paper_2606_23891_b200 import layouts
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", 0)))
    ps, cells, tasks = build_config1(sph, seed=1)
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    flush = lambda: flush_buf.fill_(1)
    sampler = ClockSampler(0)
    rows = {}
    loops = args.loops
    for name in (layouts.NAMES3 if loops == 3 else layouts.NAMES):
        w = Workload(sph, torch, ps, cells, tasks, name, loops=loops)
        t_ms = time_steps(torch, w.step, args.steps, args.warmup, flush, 1)
        g_e2e = w.capture_e2e()
        t_e2e = time_steps(torch, g_e2e.replay, args.steps, args.warmup, flush, 1)
        per = {k: [] for k, _ in w.launches()}
        for _ in range(args.steps):
            flush()
            evs = []
            for k, fn in w.launches():
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); fn(); b.record()
                evs.append((k, a, b))
            torch.cuda.synchronize()
            for k, a, b in evs:
                per[k].append(a.elapsed_time(b))
        per = {k: sum(v) / len(v) for k, v in per.items()}
        pu = sum(v for k, v in per.items() if k.startswith(("pack_", "unpack_")))
        bi, bo = w.e2e_bytes()
        rows[name] = {"substructs": [int(w.layout.stride[s]) for s in range(w.layout.n_sub)], "ms_per_step": round(sum(t_ms) / len(t_ms), 5),
                      "pack_unpack_ms": round(pu, 5), "e2e_ms_per_step": round(sum(t_e2e) / len(t_e2e), 5), "h2d_bytes_per_step": bi, "d2h_bytes_per_step": bo,
                      "kernels_ms": {k: round(v, 5) for k, v in per.items()}}
        w.close()
    clocks = sampler.stop()
    base = rows["aos"]
    for r in rows.values():
        r["pack_unpack_vs_aos"] = round(r["pack_unpack_ms"] / base["pack_unpack_ms"], 3)
        r["e2e_vs_aos"] = round(r["e2e_ms_per_step"] / base["e2e_ms_per_step"], 3)
    best = min(rows, key=lambda k: rows[k]["e2e_ms_per_step"])
    n = ps.shape[0]
    print(json.dumps({"metric": METRIC, "value": n / (rows[best]["ms_per_step"] * 1e-3), "unit": "particles/s", "n_gpus": 1, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": rows[best]["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                      "dtype": "f32", "data": "synthetic",
                      "config": {"workload": CONFIG1_NAME + ("; three-loop cycle (density, gradient, switched force)" if loops == 3 else "") + "; every particle layout of the paper",
                                 "layout": best, "loops": loops, "store": "HBM (step) / pinned host (e2e)",
                                 "l2": "flushed before every step (256 MB fill, untimed)"},
                      "e2e": {"value": n / (rows[best]["e2e_ms_per_step"] * 1e-3), "unit": "particles/s", "h2d_bytes_per_step": rows[best]["h2d_bytes_per_step"],
                              "d2h_bytes_per_step": rows[best]["d2h_bytes_per_step"]},
                      "gpu_launches": (10 if loops == 3 else 7) * args.steps, "clocks": clocks, "roofline": None, "layouts": rows}))


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def side_path():
    d = os.path.join(ROOT, "gpurun_out")
    os.makedirs(d, exist_ok=True)
    return os.path.join(d, "bench_side.json")


def compact(line, limit=4000):
    """the driver keeps only what it can parse from one stdout line: stay well below 4 KB (drop the optional keys first)"""
    for key in ("kernels", "aos", "pair_interactions_per_s", "side_file"):
        if len(json.dumps(line)) <= limit:
            break
        line.pop(key, None)
    return line


def run_default(args):
    """The default line: BASELINE.json:configs[4], the largest single-GPU configuration and the one that is the paper's whole offload
    cycle (pack, transfer, loop, transfer back, unpack; where its time goes) -- 2^26 particles, the whole
    step (density loop, ghost, force loop) in bundles of 4,096 tasks over two streams.  value = the step on an HBM-resident store;
    e2e = the same step with the store in pinned host memory, every copy inside the timed region.  One stdout line (< 4 KB);
    everything else (per-stage tables, the other configurations) goes to gpurun_out/bench_side.json."""
    import torch
    rank, world, local = dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    import paper_2606_23891_b200 as sph
    import bench_workloads as bw
    torch.cuda.set_device(local)
    hbm_peak, sm_max_mhz, peak_src = measured_peaks()
    alu_peak = N_SM * LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    common = {"hbm_peak": hbm_peak, "alu_peak": alu_peak, "peak_source": peak_src, "same_size_copy": same_size_copy_gbs, "same_size_fill": same_size_fill_gbs,
              "time_steps": lambda torch_, fn, steps, warmup, flush: time_steps(torch_, fn, steps, warmup, flush, world),
              "sampler": (lambda: ClockSampler(local)) if rank == 0 else (lambda: None)}
    t_start = time.perf_counter()
    extras = rank == 0 and world == 1 and not args.no_workloads
    R, setup, state = bw.measure_config4(args, sph, torch, common, seed=1 + rank, extras=extras)       # weak scaling: every rank owns its own box
    n = R["n"]
    ms = dist_max(R["split/resident"]["ms"], world, "cuda")
    E = R["split/staged"]
    ms_e2e = dist_max(E["ms"], world, "cuda")
    total = dist_sum(float(n), world, "cuda")
    K = R["kernel_ms"]                                                    # stage -> (ms summed over one step's launches, launches)
    dominant = max(K, key=lambda k: K[k][0])
    cand, inst, pairs = R["candidates"], R["instances"], R["neighbour_pairs"]
    flop = {"density": cand * FLOP_CAND + (pairs + n) * FLOP_HIT_DENSITY, "force": cand * FLOP_CAND + pairs * FLOP_HIT_FORCE}
    rec = {"pack_density_in": 20, "unpack_density_out": 16, "pack_force_in": 52, "unpack_force_out": 20}
    kernels = {}
    for k, (kms, cnt) in K.items():
        if k in flop:
            kernels[k] = round(flop[k] / (kms * 1e-3) / 1e12 / alu_peak, 4)
        elif k in rec:      # record bytes only: the store side of a bundle's pack / unpack (each touched cell once per launch) is left out
            kernels[k] = round(inst * rec[k] / (kms * 1e-3) / 1e9 / hbm_peak, 4)
    kms, cnt = K[dominant]
    if dominant in flop:
        roof = {"bound": "alu", "achieved": round(flop[dominant] / (kms * 1e-3) / 1e12, 3), "peak": round(alu_peak, 2), "unit": "TFLOP/s",
                "peak_source": peak_src + " max SM clock x 148 SMs x 128 FP32 lanes x 2"}
    else:
        roof = {"bound": "hbm", "achieved": round(inst * rec[dominant] / (kms * 1e-3) / 1e9, 1), "peak": hbm_peak, "unit": "GB/s",
                "peak_source": peak_src + " HBM copy bandwidth"}
    traffic = None            # dram bytes per launch of the dominant kernel from one ncu --set full capture (a committed constant, not from this run)
    tfile = os.path.join(ROOT, "profiles", "traffic_per_launch.csv")      # kernel,layout,dram_bytes_per_launch,workload
    if os.path.exists(tfile):
        for row in open(tfile):
            c = row.strip().split(",")
            if len(c) >= 4 and c[0] == dominant and c[1] == "split" and c[3] == "config4":
                traffic = float(c[2])
    roof.update(frac=round(roof["achieved"] / roof["peak"], 4), kernel=dominant, launches_per_step=cnt, launch_ms=round(kms / cnt, 4),
                share_of_step=round(kms / sum(v[0] for v in K.values()), 3), traffic=traffic,
                traffic_source="profiles/traffic_per_launch.csv (ncu --set full, r03: profiles/r03_ncu_full.md), a pair batch at full size",
                algorithmic_bytes_per_launch=round(inst * (72 if dominant == "force" else 36) / cnt),
                work="8 flop x ordered candidate pairs + 60 (force) / 25 (density) flop x pairs inside 2 h_i")
    line = {
        "metric": METRIC, "value": total / (ms * 1e-3), "unit": "particles/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": bw.CONFIG4_NAME.format(n=n), "layout": "split", "store": "HBM (value) / pinned host (e2e)",
                   "tasks": R["tasks"], "bundles": E["bundles"], "cells": setup["cells"], "l2": "inputs larger than L2 (8 GB store)", "sharding": SHARDING,
                   "timing": "one CUDA graph replay per step"},
        "pair_interactions_per_s": {"density": cand / (K["density"][0] * 1e-3), "force": cand / (K["force"][0] * 1e-3)},
        "e2e": {"value": total / (ms_e2e * 1e-3), "unit": "particles/s", "ms_per_step": ms_e2e, "h2d_bytes_per_step": E["h2d_bytes"],
                "d2h_bytes_per_step": E["d2h_bytes"],
                "path": "store in pinned host memory; density inputs up slab by slab, v and u during the density loop, results down behind the bundles; "
                        "rho, rho_dh, P, c_s, x, h, mass stay on the device between the two loops (device shadow)",
                "host_link_gbs": round((E["h2d_bytes"] + E["d2h_bytes"]) / (ms_e2e * 1e-3) / 1e9, 2),
                "link_peak_gbs": [round(R["link"]["h2d_gbs"], 1), round(R["link"]["d2h_gbs"], 1)]},
        "gpu_launches": R["split/resident"]["launches"] * args.steps, "clocks": R.get("clocks"), "roofline": roof, "kernels": kernels,
    }
    side = {"configs[4]": {"results": R, "setup": setup}}
    if "split/staged/no-shadow" in R:
        ns = R["split/staged/no-shadow"]
        line["e2e"].update(no_shadow_ms_per_step=round(ns["ms"], 3), no_shadow_bytes=[ns["h2d_bytes"], ns["d2h_bytes"]])
    if "aos/staged" in R:
        line["aos"] = {"e2e_ms_per_step": round(R["aos/staged"]["ms"], 3), "e2e_bytes": [R["aos/staged"]["h2d_bytes"], R["aos/staged"]["d2h_bytes"]],
                       "split_over_aos": round(ms_e2e / R["aos/staged"]["ms"], 3)}
    if extras:
        sub = argparse.Namespace(**vars(args))

        def attempt(name, fn):
            try:
                side[name] = fn()
            except Exception as exc:      # a failing side benchmark must not lose the headline
                side[name] = {"failed": repr(exc)}
                torch.cuda.synchronize()
            return side[name]
        sub.n = 0
        c2 = attempt("configs[2]", lambda: bw.measure_config2(sub, sph, torch, dict(common, sampler=lambda: None), seed=1)[0])
        for lay in ("split", "aos"):
            for k in ("pack_force_in", "force", "unpack_force_out"):
                try:
                    kernels[f"c2.{lay}.{k}"] = c2[lay]["kernels"][k]["frac"]
                except (KeyError, TypeError):
                    pass
        sub.steps, sub.warmup = min(args.steps, 20), 3
        attempt("configs[1]", lambda: {k: v for k, v in measure_config1(sub, sph, torch, rank, world, local).items()
                                       if k in ("value", "ms_per_step", "kernels", "aos", "e2e", "roofline")})
        sub.steps, sub.warmup, sub.n = 3, 3, args.n3
        c3 = attempt("configs[3]", lambda: bw.run_config3(sub, sph, torch, common, ks=[5, 13], modes=("streamed",)))
        for r in c3.get("sweep", []):
            kernels[f"c3.{r['layout']}.{r['op']}{r['k']}.link"] = r["moved_frac_of_link"]
        if args.full:
            sub.n, sub.steps, sub.warmup, sub.loops = 0, 5, 3, 2
            attempt("eagle-like", lambda: bw.run_eagle(sub, sph, torch, common))
            attempt("trace-replay", lambda: bw.run_replay(sub, sph, torch, common))
            attempt("cell-slots", lambda: bw.run_slots(sub, sph, torch, common))
            attempt("split-pack-loops", lambda: bw.run_fission(sub, sph, torch, common))
        if not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline_config4(state[0], budget_s=args.cpu_budget)
    if rank == 0:
        line["bench_wall_s"] = round(time.perf_counter() - t_start, 1)
        try:
            with open(side_path(), "w") as f:
                json.dump({"line": line, "side": side}, f, indent=1, default=str)
            line["side_file"] = "gpurun_out/bench_side.json"
        except OSError:
            pass
        sys.stdout.flush()
        print(json.dumps(compact(line)), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def run_ours(args):
    import torch
    if args.workload == "default":
        return run_default(args)
    if args.workload == "layouts":
        return run_layouts(args)
    if args.workload != "config1":
        return run_other_workload(args)
    rank, world, local = dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    import paper_2606_23891_b200 as sph
    torch.cuda.set_device(local)
    line = measure_config1(args, sph, torch, rank, world, local)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(budget_s=args.cpu_budget)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def measure_config1(args, sph, torch, rank, world, local):
    """configs[1]: the seven launches of a whole step (density loop then force loop), store in HBM, and the same with
    host-resident arrays; returns the JSON line as a dict"""
    hbm_peak, sm_max_mhz, peak_src = measured_peaks()
    ps, cells, tasks = build_config1(sph, seed=1 + rank)          # weak scaling: every rank owns its own box
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    flush = lambda: flush_buf.fill_(1)                            # 256 MB > 126 MB L2

    results = {}
    for name in ([args.layout] if args.layout != "both" else ["split", "aos"]):
        w = Workload(sph, torch, ps, cells, tasks, name, loops=args.loops)
        sampler = ClockSampler(local) if rank == 0 else None
        t_ms = time_steps(torch, w.step, args.steps, args.warmup, flush, world)
        clocks = sampler.stop() if sampler else None
        g_e2e = w.capture_e2e()
        t_e2e = time_steps(torch, g_e2e.replay, args.steps, args.warmup, flush, world)
        # per-kernel durations: events around each launch of each timed-length step (same stream, L2 flushed per step)
        per = {k: [] for k, _ in w.launches()}
        for _ in range(args.steps):
            flush()
            evs = []
            for k, fn in w.launches():
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); fn(); b.record()
                evs.append((k, a, b))
            torch.cuda.synchronize()
            for k, a, b in evs:
                per[k].append(a.elapsed_time(b))
        results[name] = {"w": w, "ms": sum(t_ms) / len(t_ms), "ms_e2e": sum(t_e2e) / len(t_e2e), "clocks": clocks,
                         "per": {k: sum(v) / len(v) for k, v in per.items()}}

    primary = "split" if "split" in results else args.layout
    R = results[primary]
    w = R["w"]
    ms = dist_max(R["ms"], world, "cuda")
    ms_e2e = dist_max(R["ms_e2e"], world, "cuda")
    total_particles = dist_sum(float(w.n), world, "cuda")
    alg = w.algorithmic()
    alu_peak = N_SM * LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12          # TFLOP/s at the maximum SM clock
    kernels = {}
    for k, d in R["per"].items():
        e = {"ms": round(d, 5)}
        if k in alg:
            if alg[k]["bound"] == "hbm":
                e.update(bound="hbm", achieved=round(alg[k]["bytes"] / (d * 1e-3) / 1e9, 1), peak=hbm_peak, unit="GB/s",
                         frac_of_nominal_8tbs=round(alg[k]["bytes"] / (d * 1e-3) / 1e9 / 8000.0, 4))
            else:
                e.update(bound="alu", achieved=round(alg[k]["flop"] / (d * 1e-3) / 1e12, 3), peak=round(alu_peak, 2), unit="TFLOP/s")
            e["frac"] = round(e["achieved"] / e["peak"], 4)
            if alg[k]["bound"] == "hbm":      # the same bytes as one plain copy launch on a flushed L2 (what a launch of this size can reach at all)
                e["same_size_copy_gbs"] = round(same_size_copy_gbs(torch, alg[k]["bytes"], flush), 1)
                e["frac_of_same_size_copy"] = round(e["achieved"] / e["same_size_copy_gbs"], 4)
                if k.startswith("pack_"):
                    e["same_size_fill_gbs"] = round(same_size_fill_gbs(torch, alg[k]["bytes"], flush), 1)
        kernels[k] = e
    dominant = max(R["per"], key=R["per"].get)
    traffic = None
    tfile = os.path.join(ROOT, "profiles", "traffic_per_launch.csv")      # kernel,layout,dram_bytes_per_launch,workload (from ncu --set full)
    if os.path.exists(tfile):
        for line in open(tfile):
            c = line.strip().split(",")
            if len(c) >= 4 and c[0] == dominant and c[1] == primary and c[3] == "config1":
                traffic = float(c[2])
    roof = dict(kernels[dominant])
    roof.pop("ms", None)
    roof.update(kernel=dominant, traffic=traffic, peak_source=peak_src + (" HBM copy bandwidth" if roof.get("bound") == "hbm"
                else " max SM clock x 148 SMs x 128 FP32 lanes x 2"), launch_ms=round(R["per"][dominant], 5))
    bi, bo = w.e2e_bytes()
    cand = w.info.n_candidates
    line = {
        "metric": METRIC, "value": total_particles / (ms * 1e-3), "unit": "particles/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": CONFIG1_NAME, "layout": primary, "store": "HBM", "tasks": int(w.info.n_tasks), "instances_per_loop": int(w.info.n_instances),
                   "candidate_pairs_per_loop": int(cand), "l2": "flushed before every step (256 MB fill, untimed)",
                   "sharding": SHARDING,
                   "e2e": "host-resident particle arrays; the step's copies and kernels captured once as a CUDA graph, one replay per step"},
        "pair_interactions_per_s": {"density": cand / (R["per"]["density"] * 1e-3), "force": cand / (R["per"]["force"] * 1e-3)},      # ordered candidate pairs
        "neighbour_pairs_per_s": {"density": total_particles / world * NGB_CONFIG1 / (R["per"]["density"] * 1e-3),                       # pairs inside the cut-off
                                  "force": total_particles / world * (NGB_CONFIG1 - 1) / (R["per"]["force"] * 1e-3)},
        "instances_per_s": {k: w.info.n_instances / (v * 1e-3) for k, v in R["per"].items() if k.startswith(("pack_", "unpack_"))},
        "e2e": {"value": total_particles / (ms_e2e * 1e-3), "unit": "particles/s", "h2d_bytes_per_step": bi, "d2h_bytes_per_step": bo,
                "ms_per_step": ms_e2e},
        "gpu_launches": len(w.launches()) * args.steps,
        "clocks": R["clocks"],
        "roofline": roof,
        "kernels": kernels,
    }
    for other, Ro in results.items():
        if other != primary:
            line[other] = {"value": Ro["w"].n * world / (dist_max(Ro["ms"], world, "cuda") * 1e-3), "ms_per_step": Ro["ms"],
                           "e2e_value": Ro["w"].n * world / (dist_max(Ro["ms_e2e"], world, "cuda") * 1e-3),
                           "e2e_bytes": list(Ro["w"].e2e_bytes()),
                           "kernels_ms": {k: round(v, 5) for k, v in Ro["per"].items()}}
    for Ro in results.values():
        Ro["w"].close()
    return line


# --------------------------------------------------------------------------------------------- oracle arm

def oracle_sample_step(orc, ps, cells, tasks, n_self_sample):
    """one oracle pass (pack, density, unpack, ghost, pack, force, unpack) over the tasks whose first cell is among
    the first n_self_sample cells; returns the seconds it took"""
    sel = tasks[tasks["ci"] < n_self_sample]
    t0 = time.perf_counter()
    orc.density_cycle(ps, cells, sel)
    orc.ghost(ps, float(np.float32(5.0 / 3.0)))
    orc.force_cycle(ps, cells, sel)
    return time.perf_counter() - t0


def oracle_setup():
    import oracle as orc
    import sph_inputs as si
    parts = si.config1(seed=1)
    perm, cells = orc.cells_build_grid(parts["x"], 16)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    tasks, _, _ = orc.tasks_build(cells, np.full(cells.shape[0], ps["h"].max(), dtype=np.float32))
    cores = min(os.cpu_count() or 1, 64)
    orc.set_threads(cores)
    return orc, ps, cells, tasks, cores


def oracle_stage_times(orc, ps, cells, tasks, loops=("density", "force")):
    """seconds of every stage of the oracle's cycle(s) over `tasks`, with the work each stage did"""
    out = {}
    inst = int(cells["count"][tasks["ci"]].sum() + cells["count"][tasks["cj"][tasks["cj"] >= 0]].sum())
    ni = cells["count"][tasks["ci"]].astype(np.int64)
    nj = np.where(tasks["cj"] >= 0, cells["count"][np.maximum(tasks["cj"], 0)], 0).astype(np.int64)
    cand = int(np.where(tasks["cj"] >= 0, 2 * ni * nj, ni * ni).sum())

    def timed(name, fn, work_key, work):
        t0 = time.perf_counter()
        r = fn()
        dt = time.perf_counter() - t0
        out[name] = {"s": round(dt, 4), work_key: work / dt}
        return r
    if "density" in loops:
        orc.zero(ps, orc.DENSITY_OUT)
        b_in = timed("pack_density_in", lambda: orc.pack(ps, cells, tasks, orc.DENSITY_IN), "instances_per_s", inst)
        b_out = timed("density", lambda: orc.density(cells, tasks, b_in), "candidate_pairs_per_s", cand)
        timed("unpack_density_out", lambda: orc.unpack(ps, cells, tasks, orc.DENSITY_OUT, b_out), "instances_per_s", inst)
        timed("ghost", lambda: orc.ghost(ps, float(np.float32(5.0 / 3.0))), "particles_per_s", ps.shape[0])
    if "force" in loops:
        orc.zero(ps, orc.FORCE_OUT)
        b_in = timed("pack_force_in", lambda: orc.pack(ps, cells, tasks, orc.FORCE_IN), "instances_per_s", inst)
        b_out = timed("force", lambda: orc.force(cells, tasks, b_in, 0.8, 3.0), "candidate_pairs_per_s", cand)
        timed("unpack_force_out", lambda: orc.unpack(ps, cells, tasks, orc.FORCE_OUT, b_out), "instances_per_s", inst)
    out["total_s"] = round(sum(v["s"] for v in out.values()), 4)
    return out


def oracle_config2_sample(seed=1):
    """A bounded sample of configs[2] built by the oracle's own builders: the cells of x-layers 0-3 (dense half) and 16-19
    (sparse half) of the 32^3 grid with all the tasks among them (8,192 of 32,768 cells).  h is the generator's continuum
    value (1.12725 n^-1/3, what the 48-neighbour iteration starts from), rho = m n, u from P = 1 | 0.1, P and c_s from the
    oracle's ghost: enough for timing, where only the shape of the workload matters."""
    import oracle as orc
    import sph_inputs as si
    parts = si.config2_positions(seed=seed)
    parts["h"] = np.minimum(parts["h"], np.float32(0.4999 / 32))
    perm, cells = orc.cells_build_grid(parts["x"], 32)
    ix = np.arange(cells.shape[0]) // (32 * 32)
    keep = np.flatnonzero(((ix < 4) | ((ix >= 16) & (ix < 20))) & (cells["count"] > 0))
    first, count = cells["first"].astype(np.int64), cells["count"].astype(np.int64)
    idx = np.concatenate([perm[first[c]:first[c] + count[c]] for c in keep]).astype(np.int64)
    ps = np.ascontiguousarray(parts[idx])
    sub = cells[keep].copy()
    sub["first"] = np.concatenate([[0], np.cumsum(count[keep])[:-1]])
    hmax = np.maximum.reduceat(ps["h"], sub["first"].astype(np.int64)).astype(np.float32)
    tasks, _, _ = orc.tasks_build(sub, hmax)
    n_dens = (1.12725 / ps["h"].astype(np.float64)) ** 3
    ps["rho"] = (ps["mass"] * n_dens).astype(np.float32)
    ps["u"] = (np.where(ps["x"][:, 0] < 0.5, 1.0, 0.1) / ((5.0 / 3.0 - 1.0) * ps["rho"].astype(np.float64))).astype(np.float32)
    orc.ghost(ps, float(np.float32(5.0 / 3.0)))
    return orc, ps, sub, tasks


def cpu_baseline_config2(state=None, budget_s=20.0):
    """the oracle as it stands on the host cores: the force cycle of configs[2] on a bounded sample (all threads and one thread),
    and every stage of a configs[1] step, with the CPU model"""
    orc, ps, cells, tasks = oracle_config2_sample()
    cores = min(os.cpu_count() or 1, 64)
    orc.set_threads(cores)
    # all threads: as many leading cells of the dense and of the sparse group as fit the budget
    n_cells = cells.shape[0]
    half = n_cells // 2

    def pick(m):
        ci = tasks["ci"]
        return np.ascontiguousarray(tasks[(ci < m) | ((ci >= half) & (ci < half + m))])
    probe = oracle_stage_times(orc, ps, cells, pick(128), loops=("force",))
    m = int(max(128, min(half, 128 * (0.4 * budget_s) / max(probe["total_s"], 1e-3))))
    sel = pick(m)
    st_all = oracle_stage_times(orc, ps, cells, sel, loops=("force",))
    particles = int(cells["count"][:m].sum() + cells["count"][half:half + m].sum())
    orc.set_threads(1)
    m1 = max(32, m // 8)
    st_one = oracle_stage_times(orc, ps, cells, pick(m1), loops=("force",))
    orc.set_threads(cores)
    # configs[1]: the seven stages of a whole step
    orc1, ps1, cells1, tasks1, _ = oracle_setup()
    c1_all = oracle_stage_times(orc1, ps1, cells1, tasks1)
    orc1.set_threads(1)
    c1_one = oracle_stage_times(orc1, ps1, cells1, np.ascontiguousarray(tasks1[tasks1["ci"] < 256]))
    orc1.set_threads(cores)
    return {"value": particles / st_all["total_s"], "unit": "particles/s", "cores": cores, "kind": "oracle", "cpu_model": cpu_model(),
            "hardware_concurrency": os.cpu_count(),
            "sample": f"configs[2] force cycle (pack FORCE_IN, force, unpack FORCE_OUT) over the tasks of the first {m} cells of the dense group and "
                      f"the first {m} of the sparse group of an 8192-cell sample ({particles} particles, {sel.shape[0]} tasks), {st_all['total_s']:.2f} s; "
                      f"one-thread figures on {m1} + {m1} cells; the oracle's unpack is serial by design",
            "stages": {"all_threads": st_all, "one_thread": st_one},
            "configs[1]_stages": {"all_threads_4096_cells": c1_all, "one_thread_256_cells": c1_one}}


def cpu_baseline(budget_s=20.0):
    """the oracle as it stands, on the host cores, on a bounded sample of configs[1] (about budget_s of CPU wall time):
    the tasks of the first m cells, or -- when one whole step takes less than the budget -- whole steps repeated"""
    orc, ps, cells, tasks, cores = oracle_setup()
    n_cells = cells.shape[0]
    probe = 64
    t_probe = oracle_sample_step(orc, ps, cells, tasks, probe)
    m = int(max(probe, min(n_cells, probe * budget_s / max(t_probe, 1e-3))))
    t = oracle_sample_step(orc, ps, cells, tasks, m)
    reps = 1
    if m == n_cells and t < 0.5 * budget_s:
        reps = int(max(1, min(200, budget_s / max(t, 1e-3))))
        t = sum(oracle_sample_step(orc, ps, cells, tasks, m) for _ in range(reps)) / reps
    particles = int(cells["count"][:m].sum())
    stages = oracle_stage_times(orc, ps, cells, tasks)
    return {"value": particles / t, "unit": "particles/s", "cores": cores, "kind": "oracle", "cpu_model": cpu_model(), "hardware_concurrency": os.cpu_count(),
            "sample": f"tasks of the first {m} of {n_cells} cells of configs[1] ({particles} particles), one full step, "
                      f"average of {reps} repetition(s), {t:.2f} s each", "stages": {"all_threads": stages}}


CONFIG4_SAMPLE_EDGE = 0.2     # the oracle's sample of configs[4]: the particles of the sub-cube [0, 0.2)^3 (0.8 % of the box)


def oracle_config4_sample(parts):
    """A bounded sample of the default line's input for the oracle: the particles of configs[4] (same generator, same seed, same h)
    that lie in the sub-cube [0, 0.2)^3 -- background and whatever clumps fall there -- with cells (octree, <= 400 per leaf) and
    tasks built by the oracle's own builders.  Nothing here comes from the CUDA path."""
    import oracle as orc
    inside = np.all(parts["x"] < CONFIG4_SAMPLE_EDGE, axis=1)
    sub = np.ascontiguousarray(parts[inside])
    perm, cells = orc.cells_build_octree(sub["x"], sub["h"], 400, 1.0)
    ps = np.ascontiguousarray(sub[perm.astype(np.int64)])
    tasks, _, _ = orc.tasks_build(cells, orc.cell_hmax(ps, cells), 1.0)
    return orc, ps, cells, tasks


def oracle_config4_run(parts, steps, warmup, budget_s):
    """the oracle's whole step (density cycle, ghost, force cycle) over the tasks of the first m cells of the sample, m sized so that
    warmup + steps passes take about budget_s; -> (particles per step, seconds per step, cores, sample text)"""
    orc, ps, cells, tasks = oracle_config4_sample(parts)
    cores = min(os.cpu_count() or 1, 64)
    orc.set_threads(cores)
    n_cells = cells.shape[0]
    probe = min(n_cells, 64)
    t_probe = oracle_sample_step(orc, ps, cells, tasks, probe)
    m = int(max(8, min(n_cells, probe * (budget_s / (steps + warmup)) / max(t_probe, 1e-3))))
    for _ in range(warmup):
        oracle_sample_step(orc, ps, cells, tasks, m)
    times = [oracle_sample_step(orc, ps, cells, tasks, m) for _ in range(steps)]
    particles = int(cells["count"][:m].sum())
    n_tasks = int((tasks["ci"] < m).sum())
    sample = (f"configs[4] input (same generator, seed and h), particles inside [0, {CONFIG4_SAMPLE_EDGE})^3 = {ps.shape[0]} in {n_cells} octree cells; "
              f"per step the whole cycle (pack, density, unpack, ghost, pack, force, unpack) over the {n_tasks} tasks of the first {m} cells "
              f"({particles} particles); the oracle's unpack is serial by design")
    return particles, sum(times) / len(times), cores, sample


def cpu_baseline_config4(parts, budget_s=20.0):
    particles, sec, cores, sample = oracle_config4_run(parts, steps=2, warmup=1, budget_s=budget_s)
    return {"value": particles / sec, "unit": "particles/s", "cores": cores, "kind": "oracle", "cpu_model": cpu_model(), "sample": sample}


def run_reference(args):
    """the oracle on the host cores on the default line's workload (configs[4]), each step a bounded sample of it"""
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return
    if args.workload == "config1":
        return run_reference_config1(args)
    import sph_inputs as si
    import bench_workloads as bw
    n = args.n4 or args.n or (1 << 26)
    parts = si.config4(1, n)
    particles, sec, cores, sample = oracle_config4_run(parts, args.steps, args.warmup, args.ref_budget)
    value = particles / sec
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "particles/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": bw.CONFIG4_NAME.format(n=n), "layout": "aos", "store": "host DRAM", "sample": sample},
        "cpu_baseline": {"value": value, "unit": "particles/s", "cores": cores, "kind": "oracle", "sample": sample, "cpu_model": cpu_model()},
        "e2e": {"value": value, "unit": "particles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


def run_reference_config1(args):
    orc, ps, cells, tasks, cores = oracle_setup()
    n_cells = cells.shape[0]
    probe = 32
    t_probe = oracle_sample_step(orc, ps, cells, tasks, probe)
    per_step_budget = max(0.5, args.ref_budget / (args.steps + args.warmup))
    m = int(max(8, min(n_cells, probe * per_step_budget / max(t_probe, 1e-3))))
    for _ in range(args.warmup):
        oracle_sample_step(orc, ps, cells, tasks, m)
    times = [oracle_sample_step(orc, ps, cells, tasks, m) for _ in range(args.steps)]
    particles = int(cells["count"][:m].sum())
    sec = sum(times) / len(times)
    value = particles / sec
    sample = f"tasks of the first {m} of {n_cells} cells of configs[1] ({particles} particles) per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "particles/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": CONFIG1_NAME, "layout": "aos", "store": "host DRAM", "sample": sample},
        "cpu_baseline": {"value": value, "unit": "particles/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "particles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--layout", default="both", help="split | aos | both, or any layout name of paper_2606_23891_b200/layouts.py")
    ap.add_argument("--workload", default="default", choices=["default", "config1", "config2", "config3", "config4", "link", "layouts", "eagle", "replay", "slots", "fission"],
                    help="default = configs[2] as the headline plus configs[1], [3], [4] as `workloads`; the others run one configuration "
                         "(bench_workloads.py describes them)")
    ap.add_argument("--loops", type=int, default=2, choices=[2, 3], help="layouts / config1: the two-loop cycle or the three-loop cycle (density, gradient, force)")
    ap.add_argument("--no-workloads", action="store_true", help="default line: the configs[4] headline only (split-AoS resident + staged)")
    ap.add_argument("--full", action="store_true", help="default line: also run the eagle / replay / slots / fission workloads into the side file")
    ap.add_argument("--n3", type=int, default=0, help="default line: particle count of the configs[3] entry (default 2^24)")
    ap.add_argument("--n4", type=int, default=0, help="default line: particle count of the configs[4] entry (default 2^26)")
    ap.add_argument("--n", type=int, default=0, help="particle count for config2/3/4 (default: the full size of BASELINE.json)")
    ap.add_argument("--skip-zero-copy", action="store_true", help="config4: time the staged pipeline only")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=20.0)
    ap.add_argument("--ref-budget", type=float, default=150.0, help="--impl reference: seconds of oracle work over all steps")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
