"""Workloads of bench.py beyond the default one (BASELINE.json:configs[2..4] and the host-link probe).

    python bench.py --workload config2     2^21 particles, Sod-like; pack FORCE_IN / force / unpack FORCE_OUT in bundles of 512 tasks, store in HBM
    python bench.py --workload config3     2^24 clustered particles, octree; pack-only / unpack-only sweep over 3..20 fields, store in pinned host
                                           memory, mapped zero-copy versus stage-then-H2D, AoS and split-AoS
    python bench.py --workload config4     2^26 particles, whole step streamed in bundles of 4,096 tasks over 2 streams, store in pinned host memory
    python bench.py --workload link        pinned H2D / D2H / both-ways copy bandwidth of this box (the host-link roofline)
    python bench.py --workload eagle       Eagle25-like occupancies (5 .. 125,113 per cell): whole step, every stage timed, load-balance figures
    python bench.py --workload replay      pack / unpack calls replayed from a seeded synthetic trace of offload actions, per layout
    python bench.py --workload slots       configs[1]: de-duplicated cell slots against per-task buffers (bytes, pack time, loop time)
    python bench.py --workload fission     configs[1]: the fused pack against split pack loops (by-struct / by-element / by-type), per layout

`--n N` shrinks the particle count (a power of two for config3/4, N = planes * 128 * 128 is kept for config2) for quick
runs; the default is the full size of BASELINE.json.  Everything here is harness: the path itself runs in libsph_b200.
Inputs are seeded and synthetic (sph_inputs/); no part of this file touches oracle/.
"""
import json
import math
import time

import numpy as np

from paper_2606_23891_b200.pipeline import CONFIG4_GROUP, GAMMA, Config2E2E, HostStore, Pipeline, Streamed, cell_slabs, iterate_h_on_gpu
from paper_2606_23891_b200.workloads import build_clumpy, build_config2
from sph_inputs import synthetic_trace

SWEEP_K = [3, 5, 8, 13, 16, 20]
# reading C21: the configs[3] sweeps are prefixes of these lists of 4-byte scalar components
PACK_SWEEP = [("x", 0), ("x", 1), ("x", 2), ("h", 0), ("mass", 0), ("rho", 0), ("rho_dh", 0), ("v", 0), ("v", 1), ("v", 2), ("u", 0), ("P", 0),
              ("c_s", 0), ("wcount", 0), ("wcount_dh", 0), ("a", 0), ("a", 1), ("a", 2), ("du_dt", 0), ("v_sig", 0)]
UNPACK_SWEEP = [("rho", 0), ("rho_dh", 0), ("wcount", 0), ("wcount_dh", 0), ("a", 0), ("a", 1), ("a", 2), ("du_dt", 0), ("v_sig", 0), ("div_v", 0),
                ("rot_v", 0), ("rot_v", 1), ("rot_v", 2), ("P", 0), ("c_s", 0), ("u", 0), ("v", 0), ("v", 1), ("v", 2), ("h", 0)]


def sweep_set(sph, lst, k, flags):
    return sph.make_attrset([(f, c, 1) for f, c in lst[:k]], flags)


def subs_of(sph, layout, comps):
    """substruct indices that hold the given (field, comp) list"""
    return sorted({layout.loc[sph.FIELD[f]].sub for f, _ in comps})


def ev_time(torch, fn, reps=1, stream=None):
    """milliseconds of fn() (average of reps back-to-back calls), CUDA events on the launching stream"""
    st = stream if stream is not None else torch.cuda.current_stream()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(st)
    for _ in range(reps):
        fn()
    b.record(st)
    b.synchronize()
    return a.elapsed_time(b) / reps


def timed(torch, fn, steps, warmup, before=None):
    """list of per-step ms; `before` (untimed) runs ahead of every step"""
    out = []
    for k in range(warmup + steps):
        if before:
            before()
        torch.cuda.synchronize()
        ms = ev_time(torch, fn)
        if k >= warmup:
            out.append(ms)
    return out


def link_probe(torch, nbytes=1 << 30, reps=5):
    """pinned cudaMemcpyAsync bandwidth: H2D, D2H, and both at once on two streams [GB/s of payload per direction]"""
    h_a = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    h_b = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d_a = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    d_b = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    res = {}

    def best(fn):
        t = []
        for _ in range(reps + 1):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            fn()
            torch.cuda.synchronize()
            t.append(time.perf_counter() - t0)
        return min(t[1:])

    def h2d():
        with torch.cuda.stream(s1):
            d_a.copy_(h_a, non_blocking=True)

    def d2h():
        with torch.cuda.stream(s2):
            h_b.copy_(d_b, non_blocking=True)

    res["h2d_gbs"] = nbytes / best(h2d) / 1e9
    res["d2h_gbs"] = nbytes / best(d2h) / 1e9
    res["bidir_each_gbs"] = nbytes / best(lambda: (h2d(), d2h())) / 1e9
    res["bytes"] = nbytes
    return res


# ------------------------------------------------------------------------------------------------- configs[2]

def measure_config2(args, sph, torch, common, seed=1, layouts=("split", "aos")):
    """configs[2]: per layout the whole step (pack FORCE_IN, force, unpack FORCE_OUT over 896 bundles of 512 tasks under one launch
    per stage, store in HBM), each kernel, one bundle alone, and the end-to-end step with host-resident arrays"""
    hbm_peak, alu_peak = common["hbm_peak"], common["alu_peak"]
    time_steps = common["time_steps"]
    n = args.n or (1 << 21)
    ps, cells, tasks, setup = build_config2(sph, torch, seed, n)
    n = ps.shape[0]
    params = sph.sph_params(np.float32(GAMMA), 0.8, 3.0)
    s_in, s_out = sph.sph_attrset_canonical(2), sph.sph_attrset_canonical(3)
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    flush = lambda: flush_buf.fill_(1)
    out = {}
    for name in layouts:
        layout = sph.sph_layout_split() if name == "split" else sph.sph_layout_aos()
        store = sph.sph_store_create(layout, n)
        sph.sph_store_set_cells(store, cells)
        sph.sph_store_import_aos(store, ps)
        batch = sph.sph_batch_create(store, tasks, 512)                    # 896 bundles of 512 tasks under one launch per stage
        info = sph.sph_batch_get_info(batch)
        b_in = torch.empty(sph.sph_batch_buffer_bytes(batch, s_in), dtype=torch.uint8, device="cuda")
        b_out = torch.empty(sph.sph_batch_buffer_bytes(batch, s_out), dtype=torch.uint8, device="cuda")
        # "zero the outputs" is fused into the unpack: the batch holds every task of the loop, so every particle's sums start from 0
        stages = [("pack_force_in", lambda: sph.sph_pack(store, batch, s_in, b_in)),
                  ("force", lambda: sph.sph_force(batch, b_in, b_out, params)),
                  ("unpack_force_out", lambda: sph.sph_unpack(store, batch, s_out, b_out, sph.SPH_UNPACK_REDUCE_ZERO))]
        step = lambda: [fn() for _, fn in stages]
        sampler = common["sampler"]() if name == layouts[0] else None
        t = time_steps(torch, step, args.steps, args.warmup, flush)
        clocks = sampler.stop() if sampler else None
        per = {k: [] for k, _ in stages}
        for _ in range(args.steps):
            flush()
            torch.cuda.synchronize()
            for k, fn in stages:
                per[k].append(ev_time(torch, fn))
        per = {k: sum(v) / len(v) for k, v in per.items()}
        e2e = Config2E2E(sph, torch, layout, store, batch, cells, tasks, n, (b_in, b_out), params)
        g = e2e.capture()
        t_e2e = time_steps(torch, g.replay, args.steps, args.warmup, flush)
        # one bundle alone (isolated latency of pack + force + unpack of 512 pair tasks)
        one = sph.sph_batch_create(store, tasks[info.n_self:info.n_self + 512])
        o_in = torch.empty(sph.sph_batch_buffer_bytes(one, s_in), dtype=torch.uint8, device="cuda")
        o_out = torch.empty(sph.sph_batch_buffer_bytes(one, s_out), dtype=torch.uint8, device="cuda")
        one_step = lambda: (sph.sph_pack(store, one, s_in, o_in), sph.sph_force(one, o_in, o_out, params),
                            sph.sph_unpack(store, one, s_out, o_out, sph.SPH_UNPACK_REDUCE))
        t_one = timed(torch, one_step, min(args.steps, 10), 3, before=flush)
        sph.sph_batch_destroy(one)
        inst, cand = info.n_instances, info.n_candidates
        # algorithmic bytes: every record byte once, every touched store field once per particle
        alg = {"pack_force_in": n * 64 + inst * 52, "unpack_force_out": inst * 20 + n * 20}
        # AoS moves whole 32-byte sectors of the 128-byte record (SURVEY.md 8(d)'s sector table): the pack touches all four, the
        # unpack writes two (a, du_dt in bytes 32-63; v_sig in 96-127) and DRAM fills the rest of each partially written sector
        moved = {"pack_force_in": n * 128 + inst * 52, "unpack_force_out": inst * 20 + n * (64 + 64)} if name == "aos" else None
        kern = {}
        for k, ms in per.items():
            e = {"ms": round(ms, 4)}
            if k in alg:
                e.update(bound="hbm", achieved=round(alg[k] / (ms * 1e-3) / 1e9, 1), peak=hbm_peak, unit="GB/s",
                         frac_of_nominal_8tbs=round(alg[k] / (ms * 1e-3) / 1e9 / 8000.0, 4))
                e["frac"] = round(e["achieved"] / hbm_peak, 4)
                e["instances_per_s"] = inst / (ms * 1e-3)
                if moved:
                    e["moved_bytes_sector_model"] = int(moved[k])
                    e["frac_on_moved_bytes"] = round(moved[k] / (ms * 1e-3) / 1e9 / hbm_peak, 4)
                if "same_size_copy" in common:
                    e["same_size_copy_gbs"] = round(common["same_size_copy"](torch, alg[k], flush), 1)
                    e["frac_of_same_size_copy"] = round(e["achieved"] / e["same_size_copy_gbs"], 4)
                if "same_size_fill" in common and k.startswith("pack_"):
                    e["same_size_fill_gbs"] = round(common["same_size_fill"](torch, alg[k], flush), 1)
            if k == "force":
                flop = cand * 8.0 + setup["neighbour_pairs"] * 60.0
                e.update(bound="alu", achieved=round(flop / (ms * 1e-3) / 1e12, 3), peak=round(alu_peak, 2), unit="TFLOP/s",
                         candidate_pairs_per_s=cand / (ms * 1e-3), neighbour_pairs_per_s=setup["neighbour_pairs"] / (ms * 1e-3))
                e["frac"] = round(e["achieved"] / alu_peak, 4)
            kern[k] = e
        out[name] = {"ms": sum(t) / len(t), "ms_e2e": sum(t_e2e) / len(t_e2e), "kernels": kern, "single_bundle_ms": sum(t_one) / len(t_one),
                     "tasks": int(info.n_tasks), "bundles": int(info.n_segments), "instances": int(inst), "candidate_pairs": int(cand),
                     "h2d_bytes": e2e.h2d_bytes, "d2h_bytes": e2e.d2h_bytes, "clocks": clocks, "n": n}
        e2e.close()
        sph.sph_batch_destroy(batch)
        sph.sph_store_destroy(store)
        del b_in, b_out, o_in, o_out, e2e, g
    return out, setup, (ps, cells, tasks)


CONFIG2_NAME = ("configs[2]: {n} particles, Sod-like two-density lattice (h by the 48-neighbour condition), 32^3 cells, force loop "
                "(alpha = 0.8) with pack / unpack per bundle of 512 tasks, store in HBM")


def run_config2(args, sph, torch, common):
    out, setup, _ = measure_config2(args, sph, torch, common)
    P = out["split"]
    n = P["n"]
    dominant = max(("pack_force_in", "force", "unpack_force_out"), key=lambda k: P["kernels"][k]["ms"])
    roof = {k: v for k, v in P["kernels"][dominant].items() if k != "ms"}
    roof.update(kernel=dominant, launch_ms=P["kernels"][dominant]["ms"], traffic=None)
    return {
        "value": n / (P["ms"] * 1e-3), "unit": "particles/s", "ms_per_step": P["ms"], "dtype": "f32",
        "config": {"workload": CONFIG2_NAME.format(n=n), "layout": "split", "store": "HBM", "tasks": P["tasks"], "bundles": P["bundles"],
                   "instances_per_loop": P["instances"], "candidate_pairs_per_loop": P["candidate_pairs"],
                   "l2": "flushed before every step (256 MB fill, untimed)", "setup": setup},
        "gpu_launches": 3 * args.steps, "roofline": roof, "kernels": P["kernels"], "single_bundle_ms": P["single_bundle_ms"],
        "aos": {"ms_per_step": out["aos"]["ms"], "kernels": out["aos"]["kernels"], "single_bundle_ms": out["aos"]["single_bundle_ms"],
                "e2e_ms_per_step": out["aos"]["ms_e2e"], "e2e_bytes": [out["aos"]["h2d_bytes"], out["aos"]["d2h_bytes"]]},
        "e2e": {"value": n / (P["ms_e2e"] * 1e-3), "unit": "particles/s", "h2d_bytes_per_step": P["h2d_bytes"], "d2h_bytes_per_step": P["d2h_bytes"],
                "ms_per_step": P["ms_e2e"]},
    }


# ------------------------------------------------------------------------------------------------- configs[3], configs[4]: common setup

def field_bytes(comps):
    return sum(8 if f == "x" else 4 for f, _ in comps)


def run_config3(args, sph, torch, common, ks=None, modes=("zero-copy", "staged", "streamed")):
    ks = ks or SWEEP_K
    n = args.n or (1 << 24)
    ps, cells, tasks, setup = build_clumpy(sph, 3, 1, n)
    link = link_probe(torch)
    rows = []
    best = {}
    for name in ("split", "aos"):
        layout = sph.sph_layout_split() if name == "split" else sph.sph_layout_aos()
        hs = HostStore(sph, torch, layout, ps, cells)
        dev = sph.sph_store_create(layout, n)
        sph.sph_store_set_cells(dev, cells)
        batch = sph.sph_batch_create(hs.store, tasks)
        info = sph.sph_batch_get_info(batch)
        inst = info.n_instances
        streamed = Streamed(sph, torch, cells, n_slabs=16)
        big = sweep_set(sph, PACK_SWEEP, 20, sph.SPH_ATTR_X_REL_F32)
        buf = torch.zeros(sph.sph_batch_buffer_bytes(batch, big), dtype=torch.uint8, device="cuda")
        for k in ks:
            # ---- pack
            comps = PACK_SWEEP[:k]
            aset = sweep_set(sph, PACK_SWEEP, k, sph.SPH_ATTR_X_REL_F32)
            sph.sph_batch_buffer_bytes(batch, aset)
            subs = subs_of(sph, layout, comps)
            useful = n * field_bytes(comps)                       # link-minimal: every needed store byte crosses once
            staged_bytes = sum(n * layout.stride[s] for s in subs)

            def zc():
                sph.sph_pack(hs.store, batch, aset, buf)

            def staged():
                for s in subs:
                    sph.sph_store_upload_sub(dev, s, hs.sub(s))
                sph.sph_pack(dev, batch, aset, buf)

            def streamed_p():
                streamed.pack(dev, hs, batch, aset, buf, subs)

            for mode, fn, moved in (("zero-copy", zc, None), ("staged", staged, staged_bytes), ("streamed", streamed_p, staged_bytes)):
                if mode not in modes:
                    continue
                t = min(timed(torch, fn, args.steps, min(args.warmup, 2)))
                rows.append({"op": "pack", "layout": name, "mode": mode, "k": k, "ms": round(t, 3), "particles_per_s": n / (t * 1e-3),
                             "instances_per_s": inst / (t * 1e-3), "useful_link_gbs": round(useful / (t * 1e-3) / 1e9, 2),
                             "moved_link_gbs": None if moved is None else round(moved / (t * 1e-3) / 1e9, 2),
                             "frac_of_link": round(useful / (t * 1e-3) / 1e9 / link["h2d_gbs"], 3),
                             "moved_frac_of_link": None if moved is None else round(moved / (t * 1e-3) / 1e9 / link["h2d_gbs"], 3)})
            # ---- unpack (REDUCE: += for the sums, max for v_sig, = for the rest)
            comps = UNPACK_SWEEP[:k]
            aset = sweep_set(sph, UNPACK_SWEEP, k, 0)
            sph.sph_batch_buffer_bytes(batch, aset)
            subs = subs_of(sph, layout, comps)
            useful = n * 4 * k                                    # every result field lands in the host store once
            staged_bytes = sum(n * layout.stride[s] for s in subs)

            def zc_u():
                sph.sph_unpack(hs.store, batch, aset, buf, sph.SPH_UNPACK_REDUCE)

            def staged_u():
                sph.sph_unpack(dev, batch, aset, buf, sph.SPH_UNPACK_REDUCE)
                for s in subs:
                    sph.sph_store_download_sub(dev, s, hs.sub(s))

            def streamed_u():
                streamed.unpack(dev, hs, batch, aset, buf, subs, sph.SPH_UNPACK_REDUCE)

            for mode, fn, moved in (("zero-copy", zc_u, None), ("staged", staged_u, staged_bytes), ("streamed", streamed_u, staged_bytes)):
                if mode not in modes:
                    continue
                t = min(timed(torch, fn, args.steps, min(args.warmup, 2)))
                rows.append({"op": "unpack", "layout": name, "mode": mode, "k": k, "ms": round(t, 3), "particles_per_s": n / (t * 1e-3),
                             "instances_per_s": inst / (t * 1e-3), "useful_link_gbs": round(useful / (t * 1e-3) / 1e9, 2),
                             "moved_link_gbs": None if moved is None else round(moved / (t * 1e-3) / 1e9, 2),
                             "frac_of_link": round(useful / (t * 1e-3) / 1e9 / link["d2h_gbs"], 3),
                             "moved_frac_of_link": None if moved is None else round(moved / (t * 1e-3) / 1e9 / link["d2h_gbs"], 3)})
        setup.update(tasks=int(info.n_tasks), instances=int(inst))
        sph.sph_batch_destroy(batch)
        sph.sph_store_destroy(dev)
        hs.close()
        del buf
    def pick(op, layout, k):
        c = [r for r in rows if r["op"] == op and r["layout"] == layout and r["k"] == k]
        return min(c, key=lambda r: r["ms"])
    kk = 13 if 13 in ks else ks[-1]
    p13, u13 = pick("pack", "split", kk), pick("unpack", "split", kk)
    ms = p13["ms"] + u13["ms"]
    useful13 = n * (field_bytes(PACK_SWEEP[:kk]) + 4 * kk)
    roof = {"bound": "host-link", "achieved": round(useful13 / (ms * 1e-3) / 1e9, 2), "peak": round(link["h2d_gbs"], 2), "unit": "GB/s",
            "frac": round(useful13 / (ms * 1e-3) / 1e9 / link["h2d_gbs"], 3), "traffic": None, "kernel": "pack + unpack, 13 fields, split-AoS, best mode",
            "peak_source": "pinned H2D copy bandwidth measured in this run"}
    return {"value": n / (ms * 1e-3), "unit": "particles/s", "ms_per_step": ms, "dtype": "u8",
            "config": {"workload": f"configs[3]: {n} clustered particles, octree <= 400 per leaf, pack-only / unpack-only sweep, store in pinned host memory",
                       "layout": "split", "store": "pinned host", "l2": "inputs larger than L2", "setup": setup, "link": link,
                       "step": "pack 13 fields + unpack 13 fields, each in its faster mode"},
            "gpu_launches": 2 * args.steps, "roofline": roof, "sweep": rows, "e2e": None}


# ------------------------------------------------------------------------------------------------- configs[4]



def run_config4(args, sph, torch, common, layout_names=("split", "aos")):
    n = args.n or (1 << 26)
    ps, cells, tasks, setup = build_clumpy(sph, 4, 1, n)
    n_self = int(cells.shape[0])
    link = link_probe(torch)
    res = {}
    for name in layout_names:
        layout = sph.sph_layout_split() if name == "split" else sph.sph_layout_aos()
        hs = HostStore(sph, torch, layout, ps, cells)
        for mode in ("staged", "zero-copy", "resident"):
            if mode == "zero-copy" and args.skip_zero_copy:
                continue
            if mode == "resident" and name != "split":
                continue
            pl = Pipeline(sph, torch, layout, hs, cells, tasks, n_self, 4096, mode, group=CONFIG4_GROUP)
            t0 = time.perf_counter()
            g = pl.capture()
            cap_s = time.perf_counter() - t0
            t = timed(torch, g.replay, args.steps, min(args.warmup, 2))
            ms = sum(t) / len(t)
            res[f"{name}/{mode}"] = {"ms_per_step": ms, "particles_per_s": n / (ms * 1e-3), "bundles": pl.n_bundles, "bundles_per_launch": pl.group,
                                     "launches_per_step": pl.launches,
                                     "h2d_bytes_per_step": pl.h2d_bytes, "d2h_bytes_per_step": pl.d2h_bytes,
                                     "h2d_bytes_if_no_device_shadow": pl.h2d_bytes + pl.shadow_bytes,
                                     "link_gbs": round((pl.h2d_bytes + pl.d2h_bytes) / (ms * 1e-3) / 1e9, 2) if mode == "staged" else None,
                                     "instances_per_loop": int(pl.instances), "candidate_pairs_per_loop": int(pl.candidates),
                                     "capture_s": round(cap_s, 1)}
            pl.close()
            del pl, g
        hs.close()
    key = min((k for k in res if k.startswith("split") and not k.endswith("resident")), key=lambda k: res[k]["ms_per_step"])
    P = res[key]
    compute_only = res.get("split/resident", {}).get("ms_per_step")
    link_time = max(P["h2d_bytes_per_step"] / link["h2d_gbs"], P["d2h_bytes_per_step"] / link["d2h_gbs"]) / 1e9 * 1e3 if P["h2d_bytes_per_step"] else None
    roof = {"bound": "host-link", "achieved": P["link_gbs"], "peak": round(link["h2d_gbs"], 2), "unit": "GB/s",
            "frac": None if not P["link_gbs"] else round(P["link_gbs"] / (link["h2d_gbs"] + link["d2h_gbs"]), 3), "traffic": None,
            "kernel": "whole step (H2D + pack/loop/unpack bundles + D2H)", "link_bound_ms": link_time,
            "step_over_link_time": None if not link_time else round(P["ms_per_step"] / link_time, 2),
            "compute_only_ms": compute_only,      # the same bundles on an HBM-resident store: no upload, no download
            "step_over_max_of_compute_and_link": None if not (compute_only and link_time) else round(P["ms_per_step"] / max(compute_only, link_time), 3),
            "peak_source": "pinned H2D / D2H copy bandwidth measured in this run"}
    return {"value": P["particles_per_s"], "unit": "particles/s", "ms_per_step": P["ms_per_step"], "dtype": "f32",
            "config": {"workload": f"configs[4]: {n} particles (uniform + clumps), whole step in bundles of 4096 tasks ({CONFIG4_GROUP} under one launch per stage) over 2 streams, store in pinned host memory",
                       "layout": key, "store": "pinned host", "l2": "inputs larger than L2", "setup": setup, "link": link,
                       "e2e": "staged: density inputs cross slab by slab ahead of the bundles, force inputs (v, u) during the density loop, results "
                              "behind the bundles; what the density loop and the ghost left on the device (rho, rho_dh, P, c_s; x, h, mass) is not "
                              "re-sent for the force loop (device shadow within the step; h2d_bytes_if_no_device_shadow says what it saves)"},
            "gpu_launches": P["launches_per_step"] * args.steps, "roofline": roof, "variants": res,
            "e2e": {"value": P["particles_per_s"], "unit": "particles/s", "h2d_bytes_per_step": P["h2d_bytes_per_step"],
                    "d2h_bytes_per_step": P["d2h_bytes_per_step"], "ms_per_step": P["ms_per_step"]}}


CONFIG4_NAME = ("configs[4]: {n} particles (uniform + clumps), octree cells <= 400, whole step (pack, density, unpack, ghost, pack, force, unpack) "
                "in bundles of 4096 tasks (" + str(CONFIG4_GROUP) + " under one launch per stage) over 2 streams")


def measure_config4(args, sph, torch, common, seed=1, extras=True):
    """The default line's workload.  Split-AoS: the step on an HBM-resident store (`resident`), the same step with the store in pinned
    host memory (`staged`, the end-to-end figure: copies inside the timed region), per-stage kernel times of one step; with extras
    also the staged step that keeps no device shadow between the loops, and the AoS store (staged).  Every variant is one CUDA
    graph replay per step.  Returns (results, setup, (ps, cells, tasks))."""
    n = args.n4 or args.n or (1 << 26)
    ps, cells, tasks, setup = build_clumpy(sph, 4, seed, n)
    n_self = int(cells.shape[0])
    link = link_probe(torch)
    time_steps = common["time_steps"]
    no_flush = lambda: None                      # the store (8 GB) and the buffers are far larger than L2
    res = {"n": n, "link": link}
    plan = [("split", "resident", True), ("split", "staged", True)]
    if extras:
        plan += [("split", "staged", False), ("aos", "staged", True)]
    hs, hs_name = None, None
    for name, mode, shadow in plan:
        if hs_name != name:
            if hs is not None:
                hs.close()
            layout = sph.sph_layout_split() if name == "split" else sph.sph_layout_aos()
            hs, hs_name = HostStore(sph, torch, layout, ps, cells), name
        pl = Pipeline(sph, torch, layout, hs, cells, tasks, n_self, 4096, mode, group=CONFIG4_GROUP, shadow=shadow)
        g = pl.capture()
        sampler = common["sampler"]() if (name, mode) == ("split", "resident") else None
        t = time_steps(torch, g.replay, args.steps, args.warmup, no_flush)
        key = f"{name}/{mode}" + ("" if shadow else "/no-shadow")
        res[key] = {"ms": sum(t) / len(t), "h2d_bytes": pl.h2d_bytes, "d2h_bytes": pl.d2h_bytes, "launches": pl.launches, "bundles": pl.n_bundles,
                    "batches": len(pl.batches)}
        if sampler is not None:
            res["clocks"] = sampler.stop()
        if (name, mode) == ("split", "resident"):
            res["instances"], res["candidates"], res["tasks"] = int(pl.instances), int(pl.candidates), int(tasks.shape[0])
            pl.kernel_times()                                                # warm
            res["kernel_ms"] = {k: (round(v[0], 4), v[1]) for k, v in pl.kernel_times().items()}
        if (name, mode, shadow) == ("split", "staged", True):
            # ordered pairs inside the target's own cut-off, r < 2 h_i, from the density the step has just left in the host store:
            # (32/3) pi h^3 rho / m per particle (a lower bound for the force loop, whose cut-off is max(2 h_i, 2 h_j))
            torch.cuda.synchronize()
            F = sph.FIELD
            def col(field, dtype=np.float32):
                loc = layout.loc[F[field]]
                raw = hs.host[loc.sub].numpy()[: n * layout.stride[loc.sub]].reshape(n, layout.stride[loc.sub])
                return raw[:, loc.off:loc.off + 4].copy().view(dtype).ravel().astype(np.float64)
            h, rho, m = col("h"), col("rho"), col("mass")
            ngb = (32.0 / 3.0) * np.pi * h ** 3 * rho / m
            res["neighbour_pairs"] = float(ngb.sum())
            res["neighbours_per_particle"] = float(ngb.mean())
        pl.close()
        del pl, g
    hs.close()
    return res, setup, (ps, cells, tasks)


# ------------------------------------------------------------------------------------------------- extreme occupancy, trace replay (8(f3))

def build_eagle(sph, seed, cells_per_dim, n_max=125113):
    """Eagle25-like occupancies (per cell min 5 / max 125,113 / mean 184 / median 109) on a grid of equal cells"""
    import sph_inputs as si
    parts = si.eagle_like(seed=seed, cells_per_dim=cells_per_dim, n_max=n_max)
    perm, cells = sph.sph_cells_build_grid(parts["x"], cells_per_dim)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    del parts
    hmax = np.maximum.reduceat(ps["h"], cells["first"].astype(np.int64)).astype(np.float32)
    tasks, n_self, n_pair = sph.sph_tasks_build(cells, hmax)
    cnt = cells["count"]
    info = {"particles": int(ps.shape[0]), "cells": int(cells.shape[0]), "per_cell_min": int(cnt.min()), "per_cell_max": int(cnt.max()),
            "per_cell_mean": round(float(cnt.mean()), 1), "per_cell_median": float(np.median(cnt)), "self_tasks": int(n_self), "pair_tasks": int(n_pair)}
    return ps, cells, tasks, info


def run_eagle(args, sph, torch, common):
    """whole step (density cycle, ghost, force cycle) on the extreme-occupancy set, every stage timed, AoS beside split-AoS"""
    cpd = 32 if not args.n else max(3, int(round((args.n / 190.0) ** (1.0 / 3.0))))
    ps, cells, tasks, setup = build_eagle(sph, 1, cpd)
    n = ps.shape[0]
    params = sph.sph_params(np.float32(GAMMA), 0.8, 3.0)
    sets = [sph.sph_attrset_canonical(k) for k in range(4)]
    res = {}
    for name in ("split", "aos"):
        layout = sph.sph_layout_split() if name == "split" else sph.sph_layout_aos()
        store = sph.sph_store_create(layout, n)
        sph.sph_store_set_cells(store, cells)
        sph.sph_store_import_aos(store, ps)
        batch = sph.sph_batch_create(store, tasks)
        info = sph.sph_batch_get_info(batch)
        bufs = [torch.empty(sph.sph_batch_buffer_bytes(batch, s), dtype=torch.uint8, device="cuda") for s in sets]
        Z = sph.SPH_UNPACK_REDUCE_ZERO
        stages = [("pack_density_in", lambda: sph.sph_pack(store, batch, sets[0], bufs[0])),
                  ("density", lambda: sph.sph_density(batch, bufs[0], bufs[1])),
                  ("unpack_density_out", lambda: sph.sph_unpack(store, batch, sets[1], bufs[1], Z)),
                  ("ghost", lambda: sph.sph_ghost(store, params)),
                  ("pack_force_in", lambda: sph.sph_pack(store, batch, sets[2], bufs[2])),
                  ("force", lambda: sph.sph_force(batch, bufs[2], bufs[3], params)),
                  ("unpack_force_out", lambda: sph.sph_unpack(store, batch, sets[3], bufs[3], Z))]
        step = lambda: [fn() for _, fn in stages]
        t = timed(torch, step, args.steps, min(args.warmup, 3))
        per = {k: [] for k, _ in stages}
        for _ in range(args.steps):
            torch.cuda.synchronize()
            for k, fn in stages:
                per[k].append(ev_time(torch, fn))
        per = {k: round(sum(v) / len(v), 4) for k, v in per.items()}
        inst, cand = int(info.n_instances), int(info.n_candidates)
        resident_warps = 148 * 16
        res[name] = {"ms_per_step": sum(t) / len(t), "stages_ms": per, "instances_per_loop": inst, "candidate_pairs_per_loop": cand,
                     "loop_items": int(info.n_items), "largest_item_candidates": int(info.max_item_candidates),
                     "largest_item_share_of_candidates": info.max_item_candidates / cand,
                     "largest_item_over_mean_warp_load": info.max_item_candidates / (cand / resident_warps),
                     "candidate_pairs_per_s": {"density": cand / (per["density"] * 1e-3), "force": cand / (per["force"] * 1e-3)},
                     "instances_per_s": {k: inst / (per[k] * 1e-3) for k in per if k.startswith(("pack_", "unpack_"))}}
        sph.sph_batch_destroy(batch)
        sph.sph_store_destroy(store)
        del bufs
    P = res["split"]
    return {"value": n / (P["ms_per_step"] * 1e-3), "unit": "particles/s", "ms_per_step": P["ms_per_step"], "dtype": "f32",
            "config": {"workload": f"eagle-like: {n} particles in {cpd}^3 cells of 5 .. {setup['per_cell_max']} particles (PAPER.md:164 statistics), "
                                   "density cycle, ghost, force cycle, one batch, store in HBM", "layout": "split", "store": "HBM",
                       "l2": "inputs larger than L2", "setup": setup},
            "gpu_launches": 7 * args.steps, "roofline": None, "split": P, "aos": res["aos"], "e2e": None}


def run_replay(args, sph, torch, common):
    """pack / unpack calls replayed from a synthetic trace (the spirit of SWIFTGPUPACKSIM; real traces are
    not available): one call per recorded action, no interaction loop in between, for every layout asked for"""
    from paper_2606_23891_b200 import layouts as L
    cpd = 16 if not args.n else max(3, int(round((args.n / 190.0) ** (1.0 / 3.0))))
    ps, cells, tasks, setup = build_eagle(sph, 2, cpd)
    n = ps.shape[0]
    n_self = setup["self_tasks"]
    trace = synthetic_trace(tasks.shape[0], n_self, seed=7)
    names = ["aos", "split", "pack-force", "pack-force-type"] if args.layout == "both" else [args.layout]
    sets = {("density", "pack"): sph.sph_attrset_canonical(0), ("density", "unpack"): sph.sph_attrset_canonical(1),
            ("force", "pack"): sph.sph_attrset_canonical(2), ("force", "unpack"): sph.sph_attrset_canonical(3)}
    rows = {}
    for name in names:
        layout = sph.sph_layout_aos() if name == "aos" else (sph.sph_layout_split() if name == "split" else L.layout(sph, name))
        store = sph.sph_store_create(layout, n)
        sph.sph_store_set_cells(store, cells)
        sph.sph_store_import_aos(store, ps)
        batches = {}
        need = {k: 0 for k in sets}
        inst = {"pack": 0, "unpack": 0}
        for _, loop, action, t0, m in trace:
            if (t0, m) not in batches:
                batches[(t0, m)] = sph.sph_batch_create(store, tasks[t0:t0 + m])
            b = batches[(t0, m)]
            need[(loop, action)] = max(need[(loop, action)], sph.sph_batch_buffer_bytes(b, sets[(loop, action)]))
            inst[action] += int(sph.sph_batch_get_info(b).n_instances)
        bufs = {k: torch.zeros(max(v, 256), dtype=torch.uint8, device="cuda") for k, v in need.items()}

        def replay(only=None):
            for _, loop, action, t0, m in trace:
                if only and action != only:
                    continue
                b, key = batches[(t0, m)], (loop, action)
                if action == "pack":
                    sph.sph_pack(store, b, sets[key], bufs[key])
                else:
                    sph.sph_unpack(store, b, sets[key], bufs[key], sph.SPH_UNPACK_REDUCE)
        t_all = min(timed(torch, replay, args.steps, 2))
        t_pack = min(timed(torch, lambda: replay("pack"), args.steps, 1))
        t_unpack = min(timed(torch, lambda: replay("unpack"), args.steps, 1))
        rows[name] = {"ms_all": round(t_all, 3), "ms_pack": round(t_pack, 3), "ms_unpack": round(t_unpack, 3), "calls": len(trace),
                      "pack_instances_per_s": inst["pack"] / (t_pack * 1e-3), "unpack_instances_per_s": inst["unpack"] / (t_unpack * 1e-3),
                      "us_per_call": round(1e3 * t_all / len(trace), 2)}
        for b in batches.values():
            sph.sph_batch_destroy(b)
        sph.sph_store_destroy(store)
        del bufs
    base = rows.get("aos", next(iter(rows.values())))
    for r in rows.values():
        r["vs_aos"] = round(r["ms_all"] / base["ms_all"], 3)
    best = min(rows, key=lambda k: rows[k]["ms_all"])
    total_inst = (rows[best]["pack_instances_per_s"] * rows[best]["ms_pack"] + rows[best]["unpack_instances_per_s"] * rows[best]["ms_unpack"]) * 1e-3
    return {"value": total_inst / (rows[best]["ms_all"] * 1e-3), "unit": "instances/s", "ms_per_step": rows[best]["ms_all"], "dtype": "u8",
            "metric": "particles/s packed + unpacked, trace replay",
            "config": {"workload": f"replay: synthetic trace of {len(trace)} pack / unpack actions (5 steps, bundles of 128..1024 tasks, density then force) over "
                                   f"{n} particles in {cpd}^3 cells of 5 .. {setup['per_cell_max']} particles; one call per action, no loops", "layout": best,
                       "store": "HBM", "l2": "inputs larger than L2", "setup": setup},
            "gpu_launches": len(trace) * args.steps, "roofline": None, "layouts": rows, "e2e": None}


# ------------------------------------------------------------------------------------------------- cell slots (8(f4))

def run_slots(args, sph, torch, common):
    """configs[1]: per-task buffers (a cell packed once per task side, the parity format) against de-duplicated cell slots (a cell
    packed once per batch, frames applied in the loop): bytes written by the pack, pack time, loop time, both loops"""
    import sph_inputs as si
    parts = si.config1(seed=1)
    perm, cells = sph.sph_cells_build_grid(parts["x"], 16)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    tasks, _, _ = sph.sph_tasks_build(cells, np.full(cells.shape[0], ps["h"].max(), dtype=np.float32))
    n = ps.shape[0]
    params = sph.sph_params(np.float32(GAMMA), 0.8, 3.0)
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    flush = lambda: flush_buf.fill_(1)
    layout = sph.sph_layout_split()
    store = sph.sph_store_create(layout, n)
    sph.sph_store_set_cells(store, cells)
    sph.sph_store_import_aos(store, ps)
    batch = sph.sph_batch_create(store, tasks)
    sets = [sph.sph_attrset_canonical(k) for k in range(4)]
    bufs = [torch.empty(sph.sph_batch_buffer_bytes(batch, s), dtype=torch.uint8, device="cuda") for s in sets]
    slots = [torch.empty(sph.sph_batch_slot_bytes(batch, k), dtype=torch.uint8, device="cuda") for k in range(2)]
    # physically sane inputs for the force loop
    sph.sph_pack(store, batch, sets[0], bufs[0]); sph.sph_density(batch, bufs[0], bufs[1])
    sph.sph_unpack(store, batch, sets[1], bufs[1], sph.SPH_UNPACK_REDUCE_ZERO); sph.sph_ghost(store, params)
    stages = {"pack_density_in": lambda: sph.sph_pack(store, batch, sets[0], bufs[0]),
              "pack_density_slots": lambda: sph.sph_pack_slots(store, batch, 0, slots[0]),
              "density": lambda: sph.sph_density(batch, bufs[0], bufs[1]),
              "density_slots": lambda: sph.sph_density_slots(batch, slots[0], bufs[1]),
              "pack_force_in": lambda: sph.sph_pack(store, batch, sets[2], bufs[2]),
              "pack_force_slots": lambda: sph.sph_pack_slots(store, batch, 1, slots[1]),
              "force": lambda: sph.sph_force(batch, bufs[2], bufs[3], params),
              "force_slots": lambda: sph.sph_force_slots(batch, slots[1], bufs[3], params)}
    per = {}
    for k, fn in stages.items():
        per[k] = round(sum(timed(torch, fn, args.steps, 3, before=flush)) / args.steps, 5)
    rows = {"density": {"per_task": {"input_bytes": int(bufs[0].shape[0]), "pack_ms": per["pack_density_in"], "loop_ms": per["density"]},
                        "slots": {"input_bytes": int(slots[0].shape[0]), "pack_ms": per["pack_density_slots"], "loop_ms": per["density_slots"]}},
            "force": {"per_task": {"input_bytes": int(bufs[2].shape[0]), "pack_ms": per["pack_force_in"], "loop_ms": per["force"]},
                      "slots": {"input_bytes": int(slots[1].shape[0]), "pack_ms": per["pack_force_slots"], "loop_ms": per["force_slots"]}}}
    for r in rows.values():
        r["bytes_ratio"] = round(r["per_task"]["input_bytes"] / r["slots"]["input_bytes"], 2)
        r["pack_plus_loop_ratio"] = round((r["slots"]["pack_ms"] + r["slots"]["loop_ms"]) / (r["per_task"]["pack_ms"] + r["per_task"]["loop_ms"]), 3)
    t_task = sum(per[k] for k in ("pack_density_in", "density", "pack_force_in", "force"))
    t_slot = sum(per[k] for k in ("pack_density_slots", "density_slots", "pack_force_slots", "force_slots"))
    sph.sph_batch_destroy(batch)
    sph.sph_store_destroy(store)
    return {"value": n / (t_slot * 1e-3), "unit": "particles/s", "ms_per_step": t_slot, "dtype": "f32",
            "config": {"workload": "slots: configs[1] (262144 particles, 16^3 cells), pack + loop of both loops with de-duplicated cell slots against per-task buffers",
                       "layout": "split", "store": "HBM", "l2": "flushed before every timed launch (256 MB fill, untimed)"},
            "gpu_launches": 4 * args.steps, "roofline": None, "per_task_ms": t_task, "slots_ms": t_slot, "formats": rows, "e2e": None}


def run_fission(args, sph, torch, common):
    """configs[1], pack of both loops' inputs: the fused pack kernel against the GPU analogues of the paper's split pack loops
    (Fig. 4): one pass per substruct / per quantity / per data type / per (substruct, type)"""
    import sph_inputs as si
    from paper_2606_23891_b200 import layouts as L
    parts = si.config1(seed=1)
    perm, cells = sph.sph_cells_build_grid(parts["x"], 16)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    tasks, _, _ = sph.sph_tasks_build(cells, np.full(cells.shape[0], ps["h"].max(), dtype=np.float32))
    n = ps.shape[0]
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    flush = lambda: flush_buf.fill_(1)
    names = ["aos", "split", "pack-force-type"] if args.layout == "both" else [args.layout]
    split_names = ["by-struct", "by-element", "by-type", "by-struct-and-type"]
    rows = {}
    for name in names:
        layout = L.layout(sph, name)
        store = sph.sph_store_create(layout, n)
        sph.sph_store_set_cells(store, cells)
        sph.sph_store_import_aos(store, ps)
        batch = sph.sph_batch_create(store, tasks)
        row = {}
        for label, which in (("density_in", 0), ("force_in", 2)):
            aset = sph.sph_attrset_canonical(which)
            buf = torch.empty(sph.sph_batch_buffer_bytes(batch, aset), dtype=torch.uint8, device="cuda")
            t = {"by-particle (fused)": round(min(timed(torch, lambda: sph.sph_pack(store, batch, aset, buf), args.steps, 3, before=flush)), 5)}
            passes = {}
            # the control: ONE pass of the same pass kernel with every record word selected.  The pass kernel is simple (4-byte
            # stores at record stride, no staging); the fused kernel is a tuned cp.async + bulk-copy pipeline -- so "split / fused"
            # mixes the cost of splitting with the difference between two kernels, "split / one full pass" isolates the split
            full = (1 << (sph.sph_attrset_record_bytes(aset) // 4)) - 1
            t["one full pass (same pass kernel)"] = round(min(timed(torch, lambda: sph.sph_pack_pass(store, batch, aset, full, buf), args.steps, 3, before=flush)), 5)
            for k, sname in enumerate(split_names):
                masks = sph.sph_pack_pass_masks(layout, aset, k)
                t[sname] = round(min(timed(torch, lambda: [sph.sph_pack_pass(store, batch, aset, m, buf) for m in masks], args.steps, 3, before=flush)), 5)
                passes[sname] = len(masks)
            row[label] = {"ms": t, "passes": passes, "vs_fused": {k: round(v / t["by-particle (fused)"], 2) for k, v in t.items()},
                          "vs_one_full_pass": {k: round(v / t["one full pass (same pass kernel)"], 2) for k, v in t.items()}}
            del buf
        rows[name] = row
        sph.sph_batch_destroy(batch)
        sph.sph_store_destroy(store)
    base = rows[names[0]]["force_in"]["ms"]["by-particle (fused)"]
    return {"value": n / (base * 1e-3), "unit": "particles/s", "ms_per_step": base, "dtype": "u8",
            "config": {"workload": "fission: configs[1], pack DENSITY_IN and FORCE_IN, fused kernel against one pass per substruct / quantity / data type",
                       "layout": names[0], "store": "HBM", "l2": "flushed before every timed pack (256 MB fill, untimed)"},
            "gpu_launches": args.steps, "roofline": None, "layouts": rows, "e2e": None}


def run_link(args, sph, torch, common):
    link = link_probe(torch, reps=10)
    return {"value": link["h2d_gbs"], "unit": "GB/s", "ms_per_step": None, "dtype": "u8", "metric": "pinned host-link copy bandwidth",
            "config": {"workload": "link: 1 GiB pinned cudaMemcpyAsync, best of 10", "link": link}, "gpu_launches": 0, "roofline": None, "e2e": None}


RUNNERS = {"config2": run_config2, "config3": run_config3, "config4": run_config4, "link": run_link, "eagle": run_eagle, "replay": run_replay, "slots": run_slots, "fission": run_fission}
