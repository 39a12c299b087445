"""The staging pipeline of the hot path: a particle store in pinned HOST memory streamed through the C-ABI calls on CUDA streams
("buffer contents are transferred to the GPU ... results are transferred back", PAPER.md:98 asynchronous streams).

    HostStore      the store's substruct arrays in pinned host memory (mapped: also usable zero-copy), the host side of the staged path
    cell_slabs     contiguous ranges of cells of about equal (or weighted) particle counts: the unit that crosses the host link
    Streamed       one pack or one unpack over a host-resident store, slab by slab over a copy stream and a work stream
    Pipeline       the whole step (pack, density, unpack, ghost, pack, force, unpack) in bundles of tasks over two streams, store staged
                   from / to pinned host memory (with or without a device shadow between the loops), zero-copy, or HBM-resident;
                   captured once as a CUDA graph
    Config2E2E     the force cycle of a bundle-segmented batch with host-resident arrays: slab-wise uploads and packs, the loop launched
                   per group of bundles as their cells land
    iterate_h_on_gpu   the 48-neighbour condition by Newton steps on the library's own density loop (setup of variable-h workloads)

Orchestration only: every step of the path is a call into libsph_b200 (passed in as `sph`, the binding module); torch supplies pinned
memory, streams, events and graph capture.  bench.py and the pipeline tests drive these classes; nothing here touches oracle/.
"""
import math

import numpy as np

GAMMA = float(np.float32(5.0 / 3.0))
CONFIG4_GROUP = 8      # bundles of 4,096 tasks under one launch per stage and stream (the configs[4] launch configuration)


def iterate_h_on_gpu(sph, torch, ps, cells, tasks, n_target=48.0, tol=0.01, max_iter=12):
    """48-neighbour condition (reading C20): Newton on h with wcount, wcount_dh from the library's own density loop.
    Setup for the bench workload (untimed); the parity tests use the oracle's iteration instead."""
    layout = sph.sph_layout_split()
    n = ps.shape[0]
    store = sph.sph_store_create(layout, n)
    sph.sph_store_set_cells(store, cells)
    sph.sph_store_import_aos(store, ps)
    batch = sph.sph_batch_create(store, tasks)
    s_in, s_out = sph.sph_attrset_canonical(0), sph.sph_attrset_canonical(1)
    b_in = torch.empty(sph.sph_batch_buffer_bytes(batch, s_in), dtype=torch.uint8, device="cuda")
    b_out = torch.empty(sph.sph_batch_buffer_bytes(batch, s_out), dtype=torch.uint8, device="cuda")
    h_cap = np.float32(0.4999 * cells["width"].min())
    k_n = 32.0 / 3.0 * math.pi
    sub_h, sub_o = layout.loc[sph.FIELD["h"]].sub, layout.loc[sph.FIELD["wcount"]].sub
    host_h = np.zeros((n, layout.stride[sub_h] // 4), dtype=np.float32)     # S0 = {x f64[3], h, mass}: h is word 6
    host_o = np.zeros((n, layout.stride[sub_o] // 4), dtype=np.float32)     # S1 = {rho, rho_dh, wcount, wcount_dh}
    sph.sph_store_download_sub(store, sub_h, host_h)
    torch.cuda.synchronize()
    hw = layout.loc[sph.FIELD["h"]].off // 4
    wc_w, wcd_w = layout.loc[sph.FIELD["wcount"]].off // 4, layout.loc[sph.FIELD["wcount_dh"]].off // 4
    worst = None
    for it in range(max_iter):
        sph.sph_store_zero(store, s_out)
        sph.sph_pack(store, batch, s_in, b_in)
        sph.sph_density(batch, b_in, b_out)
        sph.sph_unpack(store, batch, s_out, b_out, sph.SPH_UNPACK_REDUCE)
        sph.sph_store_download_sub(store, sub_o, host_o)
        torch.cuda.synchronize()
        h = host_h[:, hw].astype(np.float64)
        wc, wcd = host_o[:, wc_w].astype(np.float64), host_o[:, wcd_w].astype(np.float64)
        f = k_n * h ** 3 * wc - n_target
        worst = float(np.abs(f).max())
        if worst <= tol:
            break
        df = k_n * (3.0 * h ** 2 * wc + h ** 3 * wcd)
        step = np.where(df > 0, f / np.where(df > 0, df, 1.0), -0.1 * h)
        h_new = np.clip(h - step, 0.8 * h, 1.25 * h)
        host_h[:, hw] = np.minimum(h_new, h_cap).astype(np.float32)
        sph.sph_store_upload_sub(store, sub_h, host_h)
        torch.cuda.synchronize()
    out = host_h[:, hw].copy()
    sph.sph_batch_destroy(batch)
    sph.sph_store_destroy(store)
    return out, worst, it + 1


class Config2E2E:
    """configs[2] with the particle arrays in pinned HOST memory, one step = one CUDA graph:
      * the substructs the force loop reads cross slab by slab (ranges of cells) and are packed as they land (sph_pack_cells into the
        one buffer that holds all 896 bundles);
      * the slabs grow (3/16, 1/16, 1/8, 1/8, 1/4, 1/4 of the particles): the first is what the first tasks need, later ones are
        large enough to keep launches few -- the loop, not the link, sets the pace once it has started;
      * the force loop does not wait for the last slab: it runs GROUP by group of bundles (a group = a batch over a run of consecutive
        segments whose inputs are complete with the same slab; its buffers are the matching slices of the big ones, a segmented batch
        being the concatenation of its bundles' stand-alone buffers), each group as soon as that slab is packed -- so most of the loop
        overlaps the uploads; groups whose tasks reach through the periodic boundary to the far end of the cell table run last;
      * the results are reduced slab by slab (sph_unpack_cells) and each slab's particles cross back as soon as they are final."""

    def __init__(self, sph, torch, layout, store, batch, cells, tasks, n, bufs, params, fractions=(3, 1, 2, 2, 4, 4), max_segs_per_group=1 << 30, bundle=512):
        self.sph, self.torch, self.store, self.batch, self.bufs, self.params = sph, torch, store, batch, bufs, params
        F = sph.FIELD
        sub = lambda names: sorted({layout.loc[F[k]].sub for k in names})
        self.subs_in = sub(["x", "h", "mass", "rho", "rho_dh", "v", "u", "P", "c_s"])
        self.subs_out = sub(["a", "du_dt", "v_sig"])
        self.host = {s: torch.empty(n * layout.stride[s], dtype=torch.uint8).pin_memory() for s in set(self.subs_in + self.subs_out)}
        for s, h in self.host.items():
            sph.sph_store_download_sub(store, s, h)
        torch.cuda.synchronize()
        self.h2d_bytes = sum(n * layout.stride[s] for s in self.subs_in)
        self.d2h_bytes = sum(n * layout.stride[s] for s in self.subs_out)
        self.slabs = cell_slabs(cells, fractions=fractions)
        self.up, self.down = torch.cuda.Stream(), torch.cuda.Stream()
        self.loop_streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        self.s_in, self.s_out = sph.sph_attrset_canonical(2), sph.sph_attrset_canonical(3)
        # groups = runs of consecutive segments whose inputs are complete with the same slab
        _, seg_in = sph.sph_batch_block_offsets(batch, self.s_in)
        _, seg_out = sph.sph_batch_block_offsets(batch, self.s_out)
        slab_end = np.array([c0 + nc for c0, nc, _, _ in self.slabs])
        n_seg = seg_in.shape[0]
        top = np.maximum(tasks["ci"], tasks["cj"]).astype(np.int64)
        seg_top = np.maximum.reduceat(top, np.arange(0, tasks.shape[0], bundle))
        seg_need = np.searchsorted(slab_end, seg_top, side="right")
        assert seg_need.shape[0] == n_seg
        self.groups = []
        g0 = 0
        while g0 < n_seg:
            g1 = g0 + 1
            while g1 < n_seg and seg_need[g1] == seg_need[g0] and g1 - g0 < max_segs_per_group:
                g1 += 1
            gb = sph.sph_batch_create(store, tasks[g0 * bundle:min(tasks.shape[0], g1 * bundle)], bundle)
            self.groups.append({"batch": gb, "need": int(seg_need[g0]), "in": bufs[0][int(seg_in[g0]):], "out": bufs[1][int(seg_out[g0]):], "first": g0})
            g0 = g1
        self.order = sorted(range(len(self.groups)), key=lambda k: (self.groups[k]["need"], k))

    def step(self, main):
        sph, torch = self.sph, self.torch
        ev = lambda st: (lambda e: (e.record(st), e)[1])(torch.cuda.Event())
        start = ev(main)
        self.up.wait_event(start)
        self.down.wait_event(start)
        todo = list(self.order)
        for st in self.loop_streams:
            st.wait_event(start)
        n_launched = 0
        for k, (c0, nc, p0, npart) in enumerate(self.slabs):
            for s in self.subs_in:
                sph.sph_store_upload_range(self.store, s, self.host[s], p0, npart, self.up)
            main.wait_event(ev(self.up))
            sph.sph_pack_cells(self.store, self.batch, self.s_in, self.bufs[0], c0, nc, main)
            packed = ev(main)
            while todo and self.groups[todo[0]]["need"] <= k:          # every slab this group's tasks touch is packed
                g = self.groups[todo.pop(0)]
                st = self.loop_streams[n_launched & 1]                  # two streams: a group's tail overlaps the next group's start
                st.wait_event(packed)
                sph.sph_force(g["batch"], g["in"], g["out"], self.params, st)
                n_launched += 1
        assert not todo
        for st in self.loop_streams:
            main.wait_event(ev(st))
        for c0, nc, p0, npart in self.slabs:
            sph.sph_unpack_cells(self.store, self.batch, self.s_out, self.bufs[1], c0, nc, sph.SPH_UNPACK_REDUCE_ZERO, main)
            self.down.wait_event(ev(main))
            for s in self.subs_out:
                sph.sph_store_download_range(self.store, s, self.host[s], p0, npart, self.down)
        main.wait_event(ev(self.down))

    def capture(self):
        torch = self.torch
        root = torch.cuda.Stream()
        with torch.cuda.stream(root):
            self.step(root)
        torch.cuda.synchronize()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph, stream=root):
            self.step(root)
        return self.graph

    def close(self):
        self.graph = None
        for g in self.groups:
            self.sph.sph_batch_destroy(g["batch"])
        self.groups = []


class HostStore:
    """A store in pinned host memory the GPU maps (zero-copy), doubling as the host side of the staged path."""

    def __init__(self, sph, torch, layout, ps, cells):
        self.sph, self.layout, self.n = sph, layout, ps.shape[0]
        self.host = [torch.empty(sph.sph_store_sub_bytes(layout, self.n, s), dtype=torch.uint8).pin_memory() for s in range(layout.n_sub)]
        self.store = sph.sph_store_create(layout, self.n, sph.SPH_MEM_HOST_PINNED, ext=self.host)
        sph.sph_store_import_aos(self.store, ps)
        sph.sph_store_set_cells(self.store, cells)

    def sub(self, s):
        """the substruct array without its tail bytes (what upload / download move)"""
        return self.host[s][: self.n * self.layout.stride[s]]

    def close(self):
        self.sph.sph_store_destroy(self.store)
        self.host = None


def cell_slabs(cells, n_slabs=0, fractions=None):
    """[(cell_first, cell_count, particle_first, particle_count)]: contiguous cell ranges of about equal particle counts, or of the
    given relative sizes (fractions: weights, e.g. (3, 1, 2, 2, 4, 4))"""
    first = cells["first"].astype(np.int64)
    end = first + cells["count"].astype(np.int64)
    n = int(end[-1])
    if fractions is None:
        fractions = [1] * n_slabs
    cum = np.cumsum(fractions) / float(sum(fractions))
    cuts = [0]
    for k in range(len(fractions) - 1):
        c = int(np.searchsorted(end, int(cum[k] * n)))
        cuts.append(max(c, cuts[-1]))
    cuts.append(cells.shape[0])
    out = []
    for c0, c1 in zip(cuts[:-1], cuts[1:]):
        if c1 > c0:
            out.append((c0, c1 - c0, int(first[c0]), int(end[c1 - 1] - first[c0])))
    return out


class Streamed:
    """The host-resident store streamed slab by slab over two streams: the copy of slab k + 1 overlaps the kernel of slab k
    (sph_store_upload_range / sph_pack_cells, sph_unpack_cells / sph_store_download_range)."""

    def __init__(self, sph, torch, cells, n_slabs=16):
        self.sph, self.torch = sph, torch
        self.slabs = cell_slabs(cells, n_slabs)
        self.copy_s, self.work_s = torch.cuda.Stream(), torch.cuda.Stream()

    def _fork(self):
        ev = self.torch.cuda.Event()
        ev.record()
        self.copy_s.wait_event(ev)
        self.work_s.wait_event(ev)

    def _join(self):
        for st in (self.copy_s, self.work_s):
            ev = self.torch.cuda.Event()
            ev.record(st)
            self.torch.cuda.current_stream().wait_event(ev)

    def pack(self, dev, hs, batch, aset, buf, subs):
        self._fork()
        for c0, nc, p0, npart in self.slabs:
            for s in subs:
                self.sph.sph_store_upload_range(dev, s, hs.host[s], p0, npart, self.copy_s)
            ev = self.torch.cuda.Event()
            ev.record(self.copy_s)
            self.work_s.wait_event(ev)
            self.sph.sph_pack_cells(dev, batch, aset, buf, c0, nc, self.work_s)
        self._join()

    def unpack(self, dev, hs, batch, aset, buf, subs, mode):
        self._fork()
        for c0, nc, p0, npart in self.slabs:
            self.sph.sph_unpack_cells(dev, batch, aset, buf, c0, nc, mode, self.work_s)
            ev = self.torch.cuda.Event()
            ev.record(self.work_s)
            self.copy_s.wait_event(ev)
            for s in subs:
                self.sph.sph_store_download_range(dev, s, hs.host[s], p0, npart, self.copy_s)
        self._join()


class Pipeline:
    """The whole offload step streamed in bundles of `bundle` tasks over two streams, captured once as a CUDA graph.

    mode "staged" (the product path): the store lives in pinned host memory, the kernels work on a device staging store.
        * the density loop's inputs cross slab by slab (16 ranges of cells) on a copy stream; the self bundles of a slab start
          as soon as it has landed (a self task needs no other cell), the pair bundles when the last slab has;
        * pack -> loop -> unpack of a bundle run on alternating streams, unpacks chained in bundle order so the reduction order
          is the task order;
        * the force loop's extra inputs (the substructs holding v, u) cross during the density loop; what the density loop left
          on the device (rho, rho_dh, then P, c_s of the ghost) is NOT sent back up for the force loop: the device keeps it
          within the step (`shadow_bytes` says how much more the link would carry otherwise);
        * the density loop's results cross back during the force loop, the force loop's results slab by slab BEHIND the
          bundles: a cell is final once every task with ci <= cell has been unpacked.
    mode "zero-copy": the same kernels read and write the mapped host store directly over the host link.
    mode "resident": the same bundles on a store that already sits in HBM, no copies: what the step costs in kernels alone.
    """

    def __init__(self, sph, torch, layout, hs, cells, tasks, n_self, bundle, mode, n_slabs=16, group=1, shadow=True):
        """group: bundles under ONE launch per stage and stream (a batch of `group` segments of `bundle` tasks: every bundle keeps its own
        buffer slice, laid out and reduced exactly like a stand-alone bundle).
        shadow=False (staged only): SURVEY.md 8(d)'s rule for the host-resident configurations -- nothing a loop left on the device is
        used by the next one: after the ghost everything the density loop and the ghost wrote goes down to the host store, and every
        substruct the force loop reads comes up from it again, slab by slab ahead of the force bundles."""
        self.sph, self.torch, self.layout, self.hs, self.mode = sph, torch, layout, hs, mode
        self.shadow = shadow or mode != "staged"
        self.group, self.span = group, bundle * group
        n = hs.n
        self.sets = [sph.sph_attrset_canonical(k) for k in range(4)]
        self.params = sph.sph_params(np.float32(GAMMA), 0.8, 3.0)
        if mode in ("staged", "resident"):
            self.dev = sph.sph_store_create(layout, n)
            sph.sph_store_set_cells(self.dev, cells)
            self.work = self.dev
            if mode == "resident":          # the yardstick: the same bundles on a store that already sits in HBM, no copy at all
                for s_ in range(layout.n_sub):
                    sph.sph_store_upload_sub(self.dev, s_, hs.sub(s_))
                torch.cuda.synchronize()
        else:
            self.dev = None
            self.work = hs.store
        self.batches = []
        self.first_task = []          # first task of every bundle
        for lo, hi in ((0, n_self), (n_self, tasks.shape[0])):          # homogeneous bundles: self tasks, then pair tasks (C22)
            for s in range(lo, hi, self.span):
                self.batches.append(sph.sph_batch_create(hs.store, tasks[s:min(hi, s + self.span)], bundle if group > 1 else 0))
                self.first_task.append(s)
        self.n_self_bundles = sum(1 for s in self.first_task if s < n_self)
        self.n_self, self.n_tasks, self.bundle = n_self, int(tasks.shape[0]), bundle
        assert n_self == cells.shape[0] and np.all(tasks["cj"][:n_self] < 0), "the pipeline expects one self task per cell, listed first"
        self.task_ci = tasks["ci"].astype(np.int64)
        need = [0, 0, 0, 0]
        self.instances = 0
        self.candidates = 0
        self.n_bundles = sum(-(-(min(hi, s + self.span) - s) // bundle) for lo, hi in ((0, n_self), (n_self, tasks.shape[0])) for s in range(lo, hi, self.span))
        for b in self.batches:
            for k in range(4):
                need[k] = max(need[k], sph.sph_batch_buffer_bytes(b, self.sets[k]))
            info = sph.sph_batch_get_info(b)
            self.instances += info.n_instances
            self.candidates += info.n_candidates
        self.bufs = [[torch.empty(max(nb, 256), dtype=torch.uint8, device="cuda") for nb in need] for _ in range(2)]
        self.streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        self.copy = torch.cuda.Stream()
        self.slabs = cell_slabs(cells, n_slabs)                               # (cell_first, cell_count, particle_first, particle_count)
        self.slab_cell_end = np.array([c0 + nc for c0, nc, _, _ in self.slabs])
        F = sph.FIELD
        sub = lambda names: sorted({layout.loc[F[k]].sub for k in names})
        self.up_density = sub(["x", "h", "mass"])
        out_density, out_force = sub(["rho", "rho_dh", "wcount", "wcount_dh"]), sorted(set(sub(["a", "du_dt", "v_sig"]) + sub(["P", "c_s"])))
        self.up_force = [s for s in sub(["v", "u"]) if s not in self.up_density]
        self.down_force = out_force
        self.down_density = [s for s in out_density if s not in out_force]      # a substruct the force loop sends back anyway crosses once
        stride = lambda subs: sum(n * layout.stride[s] for s in subs)
        self.h2d_bytes = stride(self.up_density + self.up_force) if mode == "staged" else 0
        self.d2h_bytes = stride(self.down_density + self.down_force) if mode == "staged" else 0
        # what re-sending the force loop's inputs from the host store would add (SURVEY.md 8(d) "no device shadow across loops")
        self.shadow_bytes = stride(sorted(set(sub(["x", "h", "mass", "rho", "rho_dh", "P", "c_s"])) - set(self.up_force))) if mode == "staged" else 0
        if not self.shadow:
            self.down_mid = sorted(set(out_density + sub(["P", "c_s"])))                    # what the density loop and the ghost wrote
            self.up_force_all = sub(["x", "h", "mass", "rho", "rho_dh", "v", "u", "P", "c_s"])
            self.down_force = sub(["a", "du_dt", "v_sig"])
            self.h2d_bytes = stride(self.up_density) + stride(self.up_force_all)
            self.d2h_bytes = stride(self.down_mid) + stride(self.down_force)
        self.launches = 0

    def _bundles(self, root, k_in, k_out, kernel, slab_events):
        """pack -> loop -> unpack of every bundle on alternating streams; yields (bundle index, event of its unpack)"""
        sph, torch = self.sph, self.torch
        s_in, s_out = self.sets[k_in], self.sets[k_out]
        # "zero the outputs" is fused into the unpacks of the self bundles (every cell has exactly one self task, and the self
        # bundles come first): a cell's sums start from 0 when its self task is reduced -- after its slab has landed, which a
        # separate zero launch could not wait for in the AoS layout, where inputs and outputs share the uploaded struct
        for st in self.streams:
            st.wait_stream(root)
        prev = None
        waited_all = [False, False]
        for b, batch in enumerate(self.batches):
            st, bufs = self.streams[b & 1], self.bufs[b & 1]
            if slab_events is not None:
                if b < self.n_self_bundles:          # self tasks [t0, t1) = cells [t0, t1): wait for the slab holding the last one
                    last_cell = min(self.first_task[b] + self.span, self.n_self) - 1
                    st.wait_event(slab_events[int(np.searchsorted(self.slab_cell_end, last_cell, side="right"))])
                elif not waited_all[b & 1]:
                    st.wait_event(slab_events[-1])
                    waited_all[b & 1] = True
            sph.sph_pack(self.work, batch, s_in, bufs[k_in], st)
            kernel(batch, bufs[k_in], bufs[k_out], st)
            if prev is not None:
                st.wait_event(prev)                                       # unpacks in bundle order
            sph.sph_unpack(self.work, batch, s_out, bufs[k_out], sph.SPH_UNPACK_REDUCE_ZERO if b < self.n_self_bundles else sph.SPH_UNPACK_REDUCE, st)
            prev = torch.cuda.Event()
            prev.record(st)
            self.launches += 3
            yield b, prev
        for st in self.streams:
            root.wait_stream(st)

    def step(self, root):
        sph, torch = self.sph, self.torch
        self.launches = 0
        staged = self.mode == "staged"
        slab_events = None
        if staged:
            self.copy.wait_stream(root)
            slab_events = []
            for c0, nc, p0, npart in self.slabs:
                for s in self.up_density:
                    sph.sph_store_upload_range(self.dev, s, self.hs.host[s], p0, npart, self.copy)
                ev = torch.cuda.Event()
                ev.record(self.copy)
                slab_events.append(ev)
            for s in self.up_force:                                       # crosses during the density loop
                sph.sph_store_upload_sub(self.dev, s, self.hs.sub(s), self.copy)
            up2 = torch.cuda.Event()
            up2.record(self.copy)
        for _ in self._bundles(root, 0, 1, lambda b, i, o, st: sph.sph_density(b, i, o, st), slab_events):
            pass
        if staged:
            root.wait_event(up2)                                          # the ghost writes P, c_s next to v, u
        sph.sph_ghost(self.work, self.params, root)
        self.launches += 1
        force_slab_events = None
        if staged and self.shadow:
            self.copy.wait_stream(root)                                   # density results (and nothing the force loop writes) cross back
            for s in self.down_density:
                sph.sph_store_download_sub(self.dev, s, self.hs.sub(s), self.copy)
        elif staged:
            self.copy.wait_stream(root)                                   # no device shadow: results down, then the force loop's inputs up again
            for s in self.down_mid:
                sph.sph_store_download_sub(self.dev, s, self.hs.sub(s), self.copy)
            force_slab_events = []
            for c0, nc, p0, npart in self.slabs:
                for s in self.up_force_all:
                    sph.sph_store_upload_range(self.dev, s, self.hs.host[s], p0, npart, self.copy)
                ev = torch.cuda.Event()
                ev.record(self.copy)
                force_slab_events.append(ev)
        done_slab = 0
        for b, ev in self._bundles(root, 2, 3, lambda b, i, o, st: sph.sph_force(b, i, o, self.params, st), force_slab_events):
            if not staged or b < self.n_self_bundles:
                continue
            # every task with ci < frontier is unpacked once bundle b is: those cells are final
            nxt = self.first_task[b] + self.span
            frontier = int(self.task_ci[nxt]) if nxt < self.n_tasks else int(self.slab_cell_end[-1])
            while done_slab < len(self.slabs) and self.slab_cell_end[done_slab] <= frontier:
                _, _, p0, npart = self.slabs[done_slab]
                self.copy.wait_event(ev)
                for s in self.down_force:
                    sph.sph_store_download_range(self.dev, s, self.hs.host[s], p0, npart, self.copy)
                done_slab += 1
        if staged:
            self.copy.wait_stream(root)
            for _, _, p0, npart in self.slabs[done_slab:]:                # (only when there is no pair bundle at all)
                for s in self.down_force:
                    sph.sph_store_download_range(self.dev, s, self.hs.host[s], p0, npart, self.copy)
            root.wait_stream(self.copy)

    def capture(self):
        torch = self.torch
        root = torch.cuda.Stream()
        with torch.cuda.stream(root):
            self.step(root)                                               # warm-up outside the capture (first-call attribute setting)
        torch.cuda.synchronize()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph, stream=root):
            self.step(root)
        return self.graph

    def kernel_times(self):
        """One step launch by launch on the current stream, CUDA events around every launch (same batches, same buffers, nothing
        overlapping): {stage: (milliseconds summed over the step's launches, launches)}.  The store and buffers are far larger than
        L2, so consecutive launches do not find each other's data there."""
        sph, torch = self.sph, self.torch
        st = torch.cuda.current_stream()
        evs = []

        def timed(name, fn):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(st); fn(); b.record(st)
            evs.append((name, a, b))
        bufs = self.bufs[0]
        for loop, (k_in, k_out) in (("density", (0, 1)), ("force", (2, 3))):
            for b, batch in enumerate(self.batches):
                mode = sph.SPH_UNPACK_REDUCE_ZERO if b < self.n_self_bundles else sph.SPH_UNPACK_REDUCE
                timed(f"pack_{loop}_in", lambda: sph.sph_pack(self.work, batch, self.sets[k_in], bufs[k_in], st))
                if loop == "density":
                    timed("density", lambda: sph.sph_density(batch, bufs[0], bufs[1], st))
                else:
                    timed("force", lambda: sph.sph_force(batch, bufs[2], bufs[3], self.params, st))
                timed(f"unpack_{loop}_out", lambda: sph.sph_unpack(self.work, batch, self.sets[k_out], bufs[k_out], mode, st))
            if loop == "density":
                timed("ghost", lambda: sph.sph_ghost(self.work, self.params, st))
        torch.cuda.synchronize()
        out = {}
        for name, a, b in evs:
            ms, cnt = out.get(name, (0.0, 0))
            out[name] = (ms + a.elapsed_time(b), cnt + 1)
        return out

    def close(self):
        for b in self.batches:
            self.sph.sph_batch_destroy(b)
        if self.dev is not None:
            self.sph.sph_store_destroy(self.dev)
