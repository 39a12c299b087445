"""The configs[4] offload pipeline of bench.py (paper_2606_23891_b200.pipeline.Pipeline: bundles of 4,096 tasks over two streams, host-resident
store, streamed staging, one CUDA graph per step) against the oracle and against a plain one-stream run (needs a B200).

PAPER.md:76-82 (section 2.3: pack / launch / unpack per bundle), PAPER.md:98 (asynchronous memory streams); SURVEY.md 8(d)
"Parity at scale".  Three things are checked on a 2^19-particle instance of the configs[4] generator (6,000 octree leaves,
~25 bundles, every stream / event / slab path of the full-size run):
  * the pipeline's final HOST store equals, bit for bit, what the same kernels give when the bundles run one after the other
    on one stream against a device store (so the cross-stream unpack chain, the slab-wise uploads and the downloads behind
    the bundle frontier lose or reorder nothing);
  * that result is within the north_star tolerances of the oracle's density cycle, ghost, force cycle over the same tasks;
  * momentum and energy invariants on the pipeline's output.
"""
import numpy as np
import pytest
import torch

from paper_2606_23891_b200 import pipeline as bw, workloads
import oracle as orc
import paper_2606_23891_b200 as sph
from gpu_setup import GAMMA, PARAMS, canon
from orc_setup import raw_copy
from test_gpu_parity import check_store_physics, vsig_exempt

pytestmark = pytest.mark.gpu

_CASE = {}


def small_config4():
    if not _CASE:
        ps, cells, tasks, info = workloads.build_clumpy(sph, 4, 7, 1 << 19)
        ref = raw_copy(ps)
        orc.set_threads(64)
        oc, ot = cells.view(orc.CELL_DTYPE), tasks.view(orc.TASK_DTYPE)
        orc.density_cycle(ref, oc, ot, batch=4096)
        orc.ghost(ref, GAMMA)
        exempt = vsig_exempt(ref, oc, ot)
        orc.force_cycle(ref, oc, ot, batch=4096)
        _CASE.update(ps=ps, cells=cells, tasks=tasks, ref=ref, exempt=exempt, info=info)
    return _CASE


def one_stream_reference(layout, ps, cells, tasks, n_self, bundle):
    """the same bundles, one after the other on the current stream, store in HBM"""
    store = sph.sph_store_create(layout, ps.shape[0])
    sph.sph_store_import_aos(store, ps)
    sph.sph_store_set_cells(store, cells)
    sets = [sph.sph_attrset_canonical(k) for k in range(4)]
    batches = []
    for lo, hi in ((0, n_self), (n_self, tasks.shape[0])):
        for s in range(lo, hi, bundle):
            batches.append(sph.sph_batch_create(store, tasks[s:min(hi, s + bundle)]))
    for k_in, k_out, loop in ((0, 1, lambda b, i, o: sph.sph_density(b, i, o)), (2, 3, lambda b, i, o: sph.sph_force(b, i, o, PARAMS))):
        sph.sph_store_zero(store, sets[k_out])
        for b in batches:
            b_in = torch.empty(sph.sph_batch_buffer_bytes(b, sets[k_in]), dtype=torch.uint8, device="cuda")
            b_out = torch.empty(sph.sph_batch_buffer_bytes(b, sets[k_out]), dtype=torch.uint8, device="cuda")
            sph.sph_pack(store, b, sets[k_in], b_in)
            loop(b, b_in, b_out)
            sph.sph_unpack(store, b, sets[k_out], b_out, sph.SPH_UNPACK_REDUCE)
        if k_in == 0:
            sph.sph_ghost(store, PARAMS)
    torch.cuda.synchronize()
    out = np.zeros_like(ps)
    sph.sph_store_export_aos(store, out)
    for b in batches:
        sph.sph_batch_destroy(b)
    sph.sph_store_destroy(store)
    return out


@pytest.mark.parametrize("mode", ["staged", "zero-copy"])
@pytest.mark.parametrize("layout_name", ["split", "aos"])
def test_pipeline_equals_one_stream_run_and_oracle(layout_name, mode):
    c = small_config4()
    ps, cells, tasks, ref = c["ps"], c["cells"], c["tasks"], c["ref"]
    n_self = int(cells.shape[0])
    layout = sph.sph_layout_split() if layout_name == "split" else sph.sph_layout_aos()
    hs = bw.HostStore(sph, torch, layout, ps, cells)
    pl = bw.Pipeline(sph, torch, layout, hs, cells, tasks, n_self, 4096, mode)
    assert len(pl.batches) >= 8 and pl.n_self_bundles >= 2
    graph = pl.capture()                      # runs the step once outside the graph, then captures it
    for _ in range(2):                        # a replayed step starts from whatever the previous one left in the stores
        graph.replay()
    torch.cuda.synchronize()
    got = np.zeros_like(ps)
    sph.sph_store_export_aos(hs.store, got)
    want = one_stream_reference(layout, ps, cells, tasks, n_self, 4096)
    assert np.array_equal(canon(got), canon(want))
    check_store_physics(got, ref)
    ok = np.abs(got["v_sig"] - ref["v_sig"]) <= 1e-4 * ref["v_sig"]
    assert np.all(ok | c["exempt"]) and c["exempt"].mean() < 0.01
    m, a = got["mass"].astype(np.float64), got["a"].astype(np.float64)
    assert np.abs((m[:, None] * a).sum(0)).max() <= 1e-6 * np.abs(m[:, None] * a).sum()
    en = m * (np.einsum("ij,ij->i", got["v"].astype(np.float64), a) + got["du_dt"])
    assert abs(en.sum()) <= 1e-6 * np.abs(m * got["du_dt"].astype(np.float64)).sum()
    if mode == "staged":
        n = ps.shape[0]
        assert pl.h2d_bytes == (n * (32 + 24) if layout_name == "split" else n * 128)
        assert pl.d2h_bytes == (n * (16 + 20 + 24) if layout_name == "split" else n * 128)
    pl.close()
    hs.close()


def test_pipeline_with_grouped_bundles_equals_one_bundle_per_launch():
    """bench.py runs configs[4] with several bundles of 4,096 tasks under one launch per stage (a batch of segments): the host store
    ends up bit for bit as with one bundle per launch, which the test above ties to the one-stream run and to the oracle"""
    c = small_config4()
    ps, cells, tasks = c["ps"], c["cells"], c["tasks"]
    n_self = int(cells.shape[0])
    layout = sph.sph_layout_split()
    out = []
    for group in (1, 4):
        hs = bw.HostStore(sph, torch, layout, ps, cells)
        pl = bw.Pipeline(sph, torch, layout, hs, cells, tasks, n_self, 4096, "staged", group=group)
        assert pl.n_bundles == -(-n_self // 4096) + -(-(tasks.shape[0] - n_self) // 4096)
        pl.capture().replay()
        torch.cuda.synchronize()
        got = np.zeros_like(ps)
        sph.sph_store_export_aos(hs.store, got)
        out.append((canon(got), len(pl.batches)))
        pl.close()
        hs.close()
    assert out[1][1] < out[0][1] and np.array_equal(out[0][0], out[1][0])


@pytest.mark.parametrize("layout_name", ["split", "aos"])
def test_config2_e2e_graph_equals_plain_step(layout_name):
    """bench.py's configs[2] end-to-end step (paper_2606_23891_b200.pipeline.Config2E2E: slab-wise uploads and packs, the force loop launched per
    group of bundles as its slabs land, slab-wise unpacks and downloads, one CUDA graph) leaves in the HOST arrays exactly what the
    three plain launches leave in the store; reduced instance (31,744 particles, 8^3 cells, 14 bundles of 512 tasks)."""
    ps, cells, tasks, _ = workloads.build_config2(sph, torch, 3, 1 << 15)
    n = ps.shape[0]
    layout = sph.sph_layout_split() if layout_name == "split" else sph.sph_layout_aos()
    store = sph.sph_store_create(layout, n)
    sph.sph_store_set_cells(store, cells)
    sph.sph_store_import_aos(store, ps)
    batch = sph.sph_batch_create(store, tasks, 512)
    s_in, s_out = sph.sph_attrset_canonical(2), sph.sph_attrset_canonical(3)
    b_in = torch.empty(sph.sph_batch_buffer_bytes(batch, s_in), dtype=torch.uint8, device="cuda")
    b_out = torch.empty(sph.sph_batch_buffer_bytes(batch, s_out), dtype=torch.uint8, device="cuda")
    e2e = bw.Config2E2E(sph, torch, layout, store, batch, cells, tasks, n, (b_in, b_out), PARAMS, fractions=(1, 1, 2, 4), max_segs_per_group=3)
    assert len(e2e.groups) >= 5 and len(e2e.slabs) == 4 and sorted(e2e.order) == list(range(len(e2e.groups)))
    # the plain step
    sph.sph_pack(store, batch, s_in, b_in)
    sph.sph_force(batch, b_in, b_out, PARAMS)
    sph.sph_unpack(store, batch, s_out, b_out, sph.SPH_UNPACK_REDUCE_ZERO)
    torch.cuda.synchronize()
    want = {s: torch.empty(n * layout.stride[s], dtype=torch.uint8) for s in e2e.subs_out}
    for s, h in want.items():
        sph.sph_store_download_sub(store, s, h)
    torch.cuda.synchronize()
    assert any(int(h.view(torch.int32).abs().max()) for h in want.values())
    # the graph, from poisoned buffers and (where the substruct holds no input) poisoned host outputs
    b_in.fill_(0x7F); b_out.fill_(0x7F)
    for s in e2e.subs_out:
        if s not in e2e.subs_in:
            e2e.host[s].fill_(0x5A)
    g = e2e.capture()
    for _ in range(2):
        g.replay()
    torch.cuda.synchronize()
    for s in e2e.subs_out:
        assert torch.equal(e2e.host[s], want[s]), (layout_name, s)
    e2e.close()
    sph.sph_batch_destroy(batch)
    sph.sph_store_destroy(store)


# ------------------------------------------------------------------ bench.py's end-to-end step (host-resident arrays, three streams, one graph)

def _bench_layout_cases():
    from paper_2606_23891_b200 import layouts
    return [(n, 2) for n in layouts.NAMES] + [(n, 3) for n in layouts.NAMES3]


@pytest.mark.parametrize("name,loops", _bench_layout_cases())
def test_bench_e2e_step_equals_plain_step(name, loops):
    """bench.Workload.step_e2e (uploads, slab-wise first pack / last unpack, downloads, cross-stream events, replayed as a CUDA graph)
    leaves in the HOST mirrors exactly what the plain device-resident step leaves in the store -- for every layout, including those
    where a later loop's inputs share a substruct with an earlier loop's outputs (pack-density, pack-gradient, ...: the upload must
    be ordered before the unpack that writes that substruct).  The host mirrors start from garbage in every output field."""
    import bench
    import sph_inputs as si
    parts = si.jittered_lattice(16, seed=11)
    perm, cells = sph.sph_cells_build_grid(parts["x"], 4)
    ps = np.ascontiguousarray(parts[perm.astype(np.int64)])
    hmax = np.full(cells.shape[0], ps["h"].max(), dtype=np.float32)
    tasks, _, _ = sph.sph_tasks_build(cells, hmax)
    w = bench.Workload(sph, torch, ps, cells, tasks, name, loops=loops)
    w.step()
    torch.cuda.synchronize()
    ref = np.zeros(ps.shape[0], dtype=ps.dtype)
    sph.sph_store_export_aos(w.store, ref)
    w.close()
    dirty = ps.copy()
    rng = np.random.default_rng(5)
    for k in ("rho", "rho_dh", "wcount", "wcount_dh", "P", "c_s", "du_dt", "v_sig", "div_v"):
        dirty[k] = rng.standard_normal(ps.shape[0]).astype(np.float32)
    for k in ("a", "rot_v"):
        dirty[k] = rng.standard_normal((ps.shape[0], 3)).astype(np.float32)
    w = bench.Workload(sph, torch, dirty, cells, tasks, name, loops=loops)      # host mirrors = dirty
    g = w.capture_e2e()
    for _ in range(2):
        g.replay()
    torch.cuda.synchronize()
    # read the host mirrors back through a scratch store
    scratch = sph.sph_store_create(w.layout, ps.shape[0])
    for s_ in range(w.layout.n_sub):
        sph.sph_store_upload_sub(scratch, s_, w.host[s_])
    torch.cuda.synchronize()
    got = np.zeros(ps.shape[0], dtype=ps.dtype)
    sph.sph_store_export_aos(scratch, got)
    sph.sph_store_destroy(scratch)
    w.close()
    outs = ["rho", "rho_dh", "wcount", "wcount_dh", "P", "c_s", "a", "du_dt", "v_sig"] + (["div_v", "rot_v"] if loops == 3 else [])
    for k in outs:
        assert np.array_equal(got[k].view(np.uint32), ref[k].view(np.uint32)), (name, loops, k)
    for k in ("x", "v", "h", "mass", "u", "id", "time_bin"):
        assert np.array_equal(got[k], ps[k]), (name, loops, k)
