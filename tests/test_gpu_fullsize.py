"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (needs a B200).

configs[1] (262,144 particles, 57,344 tasks in ONE batch, exactly what `bench.py` runs): the oracle finishes a whole
step of it in about a second on the box's cores, so everything is compared in full -- pack buffers and unpack results
byte for byte, the physics of every particle within the north_star tolerances, for both store layouts.
configs[2] (2^21 particles, bundles of 512 tasks): pack FORCE_IN and unpack FORCE_OUT compared in full, byte for byte,
in the segmented launch configuration; the force loop on bundles sampled across the box (left, interface, right),
each recomputed by the oracle from the same packed records.
"""
import numpy as np
import pytest
import torch

import oracle as orc
import paper_2606_23891_b200 as sph
import sph_inputs as si
from gpu_setup import GAMMA, PARAMS, GpuCase, canon, to_attrset, valid_mask
from orc_setup import raw_copy, sort_grid
from test_gpu_parity import _random_result_buffer, _records, check_store_physics, gpu_step

pytestmark = pytest.mark.gpu

_C1 = {}


def config1():
    if not _C1:
        orc.set_threads(64)
        ps, cells, tasks, n_self, n_pair = sort_grid(si.config1(seed=1), 16)
        assert (n_self, n_pair) == (4096, 53248) and np.all(cells["count"] == 64)
        ref = raw_copy(ps)
        orc.density_cycle(ref, cells, tasks)
        orc.ghost(ref, GAMMA)
        orc.force_cycle(ref, cells, tasks)
        _C1.update(ps=ps, cells=cells, tasks=tasks, ref=ref)
    return _C1["ps"], _C1["cells"], _C1["tasks"], _C1["ref"]


def _block_mask(cells, tasks, rec, total):
    """bytes of a buffer that blocks occupy, vectorised (pad bytes are unspecified)"""
    off, tot = orc.block_offsets(cells, tasks, rec)
    assert tot == total
    m = np.zeros(total + 1, dtype=np.int32)
    for side, key in ((0, "ci"), (1, "cj")):
        c = tasks[key].astype(np.int64)
        sel = c >= 0
        o = off[side::2][sel].astype(np.int64)
        n = cells["count"][c[sel]].astype(np.int64) * rec
        np.add.at(m, o, 1)
        np.add.at(m, o + n, -1)
    return np.cumsum(m[:-1]) > 0


@pytest.mark.parametrize("layout", ["split", "aos"])
def test_config1_whole_step_every_particle(layout):
    ps, cells, tasks, ref = config1()
    g = GpuCase(ps, cells, tasks, layout)                # one batch holding every task, zeroing fused into the unpacks: bench.py's configuration
    got = gpu_step(g, fused_zero=True)
    sph.sph_store_import_aos(g.store, ps)
    assert np.array_equal(canon(gpu_step(g)), canon(got))      # the seven-launch step equals the nine-launch one bit for bit
    check_store_physics(got, ref)
    vs_ok = np.abs(got["v_sig"] - ref["v_sig"]) <= 1e-4 * ref["v_sig"]
    assert vs_ok.mean() > 0.999                          # C31: only particles with a neighbour on the cut-off may differ
    for fld in ("x", "v", "mass", "h", "u", "div_v", "rot_v", "id", "time_bin"):
        assert np.array_equal(got[fld], ps[fld]), fld
    m = got["mass"].astype(np.float64)
    a = got["a"].astype(np.float64)
    assert np.abs((m[:, None] * a).sum(0)).max() <= 1e-6 * np.abs(m[:, None] * a).sum()
    g.close()


@pytest.mark.parametrize("layout", ["split", "aos"])
def test_config1_pack_and_unpack_bytes_in_full(layout):
    ps, cells, tasks, ref = config1()
    filled = raw_copy(ref)                               # physically consistent values in every field the sets touch
    g = GpuCase(filled, cells, tasks, layout)
    for oset in (orc.DENSITY_IN, orc.FORCE_IN):
        want = orc.pack(filled, cells, tasks, oset)
        buf = g.pack(to_attrset(oset)).cpu().numpy()
        mask = _block_mask(cells, tasks, orc.record_bytes(oset), want.shape[0])
        assert buf.shape == want.shape and np.array_equal(buf[mask], want[mask])
    for n_set, oset in enumerate((orc.DENSITY_OUT, orc.FORCE_OUT)):
        rec = orc.record_bytes(oset)
        _, total = orc.block_offsets(cells, tasks, rec)
        res = _random_result_buffer(total, 300 + n_set)
        want = raw_copy(filled)
        orc.unpack(want, cells, tasks, oset, res, orc.MODE_REDUCE)
        sph.sph_store_import_aos(g.store, filled)
        sph.sph_unpack(g.store, g.batch, to_attrset(oset), torch.from_numpy(res).cuda(), sph.SPH_UNPACK_REDUCE)
        assert np.array_equal(canon(g.export()), canon(want)), rec
    g.close()


def test_config1_loops_every_record():
    """density and force result buffers of the one-batch launch, every record of every task side"""
    ps, cells, tasks, ref = config1()
    g = GpuCase(ref, cells, tasks, "split")
    b_in = orc.pack(ref, cells, tasks, orc.DENSITY_IN)
    want = orc.density(cells, tasks, b_in)
    d_out = g.buffer(to_attrset(orc.DENSITY_OUT))
    sph.sph_density(g.batch, torch.from_numpy(b_in).cuda(), d_out)
    torch.cuda.synchronize()
    got = d_out.cpu().numpy()
    mask = _block_mask(cells, tasks, 16, want.shape[0])
    w4, g4 = want[mask].view(np.float32).reshape(-1, 4).astype(np.float64), got[mask].view(np.float32).reshape(-1, 4).astype(np.float64)
    h = float(ref["h"][0])
    mass = float(ref["mass"][0])
    # partial sums of one task side: tolerances relative to the scale of a full sum (C32), as in test_gpu_parity
    scale = np.array([mass, mass / h, 1.0, 1.0 / h]) / (np.pi * h ** 3)
    assert np.all(np.abs(g4 - w4) <= 2e-5 * np.maximum(np.abs(w4), scale))
    f_in = orc.pack(ref, cells, tasks, orc.FORCE_IN)
    want = orc.force(cells, tasks, f_in, 0.8, 3.0)
    f_out = g.buffer(to_attrset(orc.FORCE_OUT))
    sph.sph_force(g.batch, torch.from_numpy(f_in).cuda(), f_out, PARAMS)
    torch.cuda.synchronize()
    got = f_out.cpu().numpy()
    mask = _block_mask(cells, tasks, 20, want.shape[0])
    w5, g5 = want[mask].view(np.float32).reshape(-1, 5).astype(np.float64), got[mask].view(np.float32).reshape(-1, 5).astype(np.float64)
    amax, dumax = np.abs(ref["a"]).max(), np.abs(ref["du_dt"]).max()
    assert np.all(np.abs(g5[:, :3] - w5[:, :3]) <= np.maximum(1e-4 * np.abs(w5[:, :3]), 1e-6 * amax))
    assert np.all(np.abs(g5[:, 3] - w5[:, 3]) <= np.maximum(1e-4 * np.abs(w5[:, 3]), 1e-6 * dumax))
    assert (np.abs(g5[:, 4] - w5[:, 4]) <= 1e-4 * np.abs(w5[:, 4])).mean() > 0.999
    g.close()


# ------------------------------------------------------------------ configs[2]

_C2 = {}


def config2():
    """2^21 particles of the Sod-like setup in cell order with seeded (not iterated) variable h: the byte-level checks
    need only the shape of the workload (102 / 26 particles per cell, bundles of 512), not converged physics."""
    if not _C2:
        orc.set_threads(64)
        parts = si.config2_positions(seed=1)
        ps, cells, tasks, n_self, n_pair = sort_grid(parts, 32)
        assert ps.shape[0] == 1 << 21 and n_self == 32768
        rng = np.random.default_rng(5)
        for name in ("v",):
            ps[name] = (0.1 * rng.standard_normal((ps.shape[0], 3))).astype(np.float32)
        for name in ("rho", "P", "c_s", "u"):
            ps[name] = (rng.random(ps.shape[0]) + 0.5).astype(np.float32)
        ps["rho_dh"] = (rng.standard_normal(ps.shape[0]) * 0.1).astype(np.float32)
        _C2.update(ps=ps, cells=cells, tasks=tasks)
    return _C2["ps"], _C2["cells"], _C2["tasks"]


def test_config2_pack_unpack_bundles_of_512_bytes_in_full():
    ps, cells, tasks = config2()
    g = GpuCase(ps, cells, tasks, "split", tasks_per_segment=512)      # 64 + 832 bundles under one launch: bench.py --workload config2
    info = sph.sph_batch_get_info(g.batch)
    assert info.n_segments == 896
    aset = to_attrset(orc.FORCE_IN)
    got = g.pack(aset).cpu().numpy()
    off, seg_off = sph.sph_batch_block_offsets(g.batch, aset)
    # bundle by bundle the oracle packs the bundle's tasks as a stand-alone batch; compare a spread of bundles in full
    for b in list(range(0, 896, 37)) + [63, 64, 895]:
        sel = tasks[512 * b:512 * (b + 1)]
        want = orc.pack(ps, cells, sel, orc.FORCE_IN)
        mask = _block_mask(cells, sel, 52, want.shape[0])
        lo = int(seg_off[b])
        assert np.array_equal(got[lo:lo + want.shape[0]][mask], want[mask]), b
    # unpack of the whole segmented buffer against the oracle run bundle after bundle (ascending task order)
    rec = 20
    oset = orc.FORCE_OUT
    aset = to_attrset(oset)
    total = sph.sph_batch_buffer_bytes(g.batch, aset)
    res = _random_result_buffer(total, 77)
    _, seg_off = sph.sph_batch_block_offsets(g.batch, aset)
    want = raw_copy(ps)
    for b in range(896):
        sel = tasks[512 * b:512 * (b + 1)]
        _, tot_b = orc.block_offsets(cells, sel, rec)
        lo = int(seg_off[b])
        orc.unpack(want, cells, sel, oset, res[lo:lo + tot_b], orc.MODE_REDUCE)
    sph.sph_unpack(g.store, g.batch, aset, torch.from_numpy(res).cuda(), sph.SPH_UNPACK_REDUCE)
    assert np.array_equal(canon(g.export()), canon(want))
    g.close()


def test_config2_force_on_sampled_bundles():
    ps, cells, tasks = config2()
    ps = raw_copy(ps)
    ps["rho"] = np.where(ps["x"][:, 0] < 0.5, 1.568, 0.4).astype(np.float32)      # plausible densities of the two halves
    ps["rho_dh"] = 0
    g = GpuCase(ps, cells, tasks, "split", tasks_per_segment=512)
    s_in, s_out = to_attrset(orc.FORCE_IN), to_attrset(orc.FORCE_OUT)
    b_in = g.pack(s_in)
    b_out = g.buffer(s_out)
    sph.sph_force(g.batch, b_in, b_out, PARAMS)
    torch.cuda.synchronize()
    got_in, got_out = b_in.cpu().numpy(), b_out.cpu().numpy()
    _, seg_in = sph.sph_batch_block_offsets(g.batch, s_in)
    _, seg_out = sph.sph_batch_block_offsets(g.batch, s_out)
    for b in (0, 40, 64, 100, 470, 480, 800, 895):       # self bundles, pair bundles left / at the interface / right
        sel = tasks[512 * b:512 * (b + 1)]
        want_in = orc.pack(ps, cells, sel, orc.FORCE_IN)
        want = orc.force(cells, sel, want_in, 0.8, 3.0)
        mask = _block_mask(cells, sel, 20, want.shape[0])
        lo = int(seg_out[b])
        w5 = want[mask].view(np.float32).reshape(-1, 5).astype(np.float64)
        g5 = got_out[lo:lo + want.shape[0]][mask].view(np.float32).reshape(-1, 5).astype(np.float64)
        amax, dumax = np.abs(w5[:, :3]).max(), np.abs(w5[:, 3]).max()
        assert np.all(np.abs(g5[:, :3] - w5[:, :3]) <= np.maximum(1e-4 * np.abs(w5[:, :3]), 1e-6 * amax)), b
        assert np.all(np.abs(g5[:, 3] - w5[:, 3]) <= np.maximum(1e-4 * np.abs(w5[:, 3]), 1e-6 * dumax)), b
        assert (np.abs(g5[:, 4] - w5[:, 4]) <= 1e-4 * np.abs(w5[:, 4]) + 1e-30).mean() > 0.995, b
    g.close()
