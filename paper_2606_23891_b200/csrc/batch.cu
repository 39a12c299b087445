// Batches ("bundles"): the immutable device tables every kernel of the hot path indexes.
#include <algorithm>
#include <cstring>
#include <memory>

#include "internal.h"

using namespace sph;

namespace {

template <class T>
int32_t upload(const std::vector<T>& v, T** d) {
    *d = nullptr;
    if (v.empty()) return SPH_OK;
    cudaError_t e = cudaMalloc((void**)d, v.size() * sizeof(T));
    if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? SPH_ERR_ALLOC : SPH_ERR_CUDA, "cudaMalloc(%zu): %s", v.size() * sizeof(T), cudaGetErrorString(e));
    e = cudaMemcpy(*d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return fail(SPH_ERR_CUDA, "cudaMemcpy: %s", cudaGetErrorString(e));
    return SPH_OK;
}

struct BatchDeleter { void operator()(sph_batch* b) const { sph_batch_destroy(b); } };

}  // namespace

namespace sph {

// Block offsets for one record size: every block starts at the next multiple of 128 bytes, every segment at
// the next multiple of 256 bytes (a segment is laid out exactly like a stand-alone batch of its tasks).
// Built the first time a record size is used (any thread), found afterwards; the batch's other tables never change.
int32_t ensure_offsets(const sph_batch* b, uint32_t rec_bytes, const OffsetTable** out) {
    std::lock_guard<std::mutex> lock(b->mu);
    auto it = b->offsets.find(rec_bytes);
    if (it != b->offsets.end()) { if (out) *out = &it->second; return SPH_OK; }
    OffsetTable ot;
    ot.h_off.resize(b->n_sides);
    std::vector<uint32_t> off128(b->n_sides);
    uint64_t run = 0;
    const uint64_t tps = b->tasks_per_segment ? b->tasks_per_segment : b->n_tasks;
    for (uint64_t t = 0; t < b->n_tasks; ++t) {
        if (t % tps == 0) { run = (run + 255) / 256 * 256; ot.seg_off.push_back(run); }
        for (uint32_t s = b->task_side0[t]; s < b->task_side0[t + 1]; ++s) {
            ot.h_off[s] = run;
            off128[s] = (uint32_t)(run / 128);
            run = (run + (uint64_t)b->sides[s].count * rec_bytes + 127) / 128 * 128;
        }
    }
    ot.total = run;
    if (run / 128 >= (1ull << 32)) return fail(SPH_ERR_RANGE, "buffer of %llu bytes exceeds the 512 GiB offset range", (unsigned long long)run);
    if (int32_t rc = upload(off128, &ot.d_off128)) return rc;
    std::vector<uint32_t> occ_off128(b->occ_side.size());
    for (size_t o = 0; o < occ_off128.size(); ++o) occ_off128[o] = off128[b->occ_side[o]];
    if (int32_t rc = upload(occ_off128, &ot.d_occ_off128)) { cudaFree(ot.d_off128); return rc; }
    auto ins = b->offsets.emplace(rec_bytes, std::move(ot));
    if (out) *out = &ins.first->second;
    return SPH_OK;
}

// Slot tables of one loop: every touched cell gets one slot of `count` records (x raw f64, so the frame can be applied in
// the loop exactly as the pack applies it: (float)(x - frame)), slots in ascending cell index, each starting at a multiple of
// 128 bytes; the loop's items are the batch's items with their record offsets pointing into the slot buffer.
int32_t ensure_slots(const sph_batch* b, int loop, const SlotTables** out) {
    if (loop < 0 || loop > 1) return fail(SPH_ERR_INVALID_ARG, "loop must be 0 (density) or 1 (force)");
    std::lock_guard<std::mutex> lock(b->mu);
    SlotTables& sl = b->slots[loop];
    if (sl.built) { *out = &sl; return SPH_OK; }
    const uint32_t rec = loop == 0 ? 36u : 68u, out_rec = loop == 0 ? 16u : 20u;
    const uint32_t n_cells = (uint32_t)b->cell_chunk0.size() - 1;
    std::vector<uint32_t> cell_first(n_cells, 0), cell_count(n_cells, 0);
    std::vector<char> touched(n_cells, 0);
    for (const SideRec& s : b->sides) { touched[s.cell] = 1; cell_first[s.cell] = s.first; cell_count[s.cell] = s.count; }
    std::vector<uint32_t> slot128(n_cells, 0), off128;
    std::vector<CellChunk> chunks;
    uint64_t run = 0;
    uint32_t idx = 0;
    for (uint32_t c = 0; c < n_cells; ++c) {
        if (!touched[c]) continue;
        slot128[c] = (uint32_t)(run / 128);
        off128.push_back(slot128[c]);
        for (uint32_t k = 0; k < cell_count[c]; k += 32) chunks.push_back(CellChunk{cell_first[c] + k, std::min(32u, cell_count[c] - k), k, idx, 1u});
        run = (run + (uint64_t)cell_count[c] * rec + 127) / 128 * 128;
        ++idx;
    }
    if (run / 128 >= (1ull << 32)) return fail(SPH_ERR_RANGE, "slot buffer exceeds the 512 GiB offset range");
    auto it = b->offsets.find(out_rec);
    if (it == b->offsets.end()) return fail(SPH_ERR_INVALID_ARG, "batch has no result offsets");
    const std::vector<uint64_t>& oout = it->second.h_off;
    std::vector<LoopItem> items(b->item_side.size());
    std::vector<double> ifr(6 * b->item_side.size());
    for (size_t i = 0; i < items.size(); ++i) {
        const ItemSide& is = b->item_side[i];
        const SideRec &t = b->sides[is.tgt], &s = b->sides[is.src];
        items[i] = LoopItem{slot128[t.cell] + is.kc * 2 * (rec / 4), slot128[s.cell], (uint32_t)(oout[is.tgt] / 128) + is.kc * 2 * (out_rec / 4),
                            std::min(kLoopTargets, t.count - is.kc * kLoopTargets) | s.count << 7};
        std::copy_n(&b->side_frames[3 * (size_t)is.tgt], 3, &ifr[6 * i]);
        std::copy_n(&b->side_frames[3 * (size_t)is.src], 3, &ifr[6 * i + 3]);
    }
    std::vector<double> zeros(3 * (size_t)idx, 0.0);
    // upload straight into the batch's tables: if one upload fails, sph_batch_destroy frees the arrays made so far and
    // a later call starts over (`built` is set last)
    auto drop = [&](int32_t rc) {
        cudaFree(sl.d_chunks); cudaFree(sl.d_slot_off128); cudaFree(sl.d_zero_frames); cudaFree(sl.d_items); cudaFree(sl.d_item_frames);
        sl = SlotTables{};
        return rc;
    };
    if (int32_t rc = upload(chunks, &sl.d_chunks)) return drop(rc);
    if (int32_t rc = upload(off128, &sl.d_slot_off128)) return drop(rc);
    if (int32_t rc = upload(zeros, &sl.d_zero_frames)) return drop(rc);
    if (int32_t rc = upload(items, &sl.d_items)) return drop(rc);
    if (int32_t rc = upload(ifr, &sl.d_item_frames)) return drop(rc);
    sl.rec_bytes = rec; sl.total = run; sl.n_chunks = (uint32_t)chunks.size(); sl.built = true;
    *out = &sl;
    return SPH_OK;
}

}  // namespace sph

extern "C" {

int32_t sph_batch_create(const sph_store* store, const sph_task* tasks, uint64_t n_tasks, uint32_t tasks_per_segment, sph_batch** out) {
    if (!out) return fail(SPH_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!store || !tasks || n_tasks == 0) return fail(SPH_ERR_INVALID_ARG, "store or tasks is NULL, or no tasks");
    if (store->cells.empty()) return fail(SPH_ERR_INVALID_ARG, "the store has no cell table (sph_store_set_cells)");
    if (n_tasks >= (1ull << 30)) return fail(SPH_ERR_RANGE, "too many tasks (%llu; side indices are 32-bit)", (unsigned long long)n_tasks);
    SPH_API_BEGIN
    const uint32_t n_cells = (uint32_t)store->cells.size();
    std::unique_ptr<sph_batch, BatchDeleter> holder(new sph_batch());
    sph_batch* b = holder.get();
    b->n_tasks = n_tasks;
    b->store_n = store->n;
    b->cells_hash = store->cells_hash;
    b->tasks_per_segment = tasks_per_segment;
    b->n_segments = tasks_per_segment ? (uint32_t)((n_tasks + tasks_per_segment - 1) / tasks_per_segment) : 1;
    std::vector<double> frames;
    std::vector<uint32_t> partner;            // per side: the side its targets gather from
    b->task_side0.resize(n_tasks + 1);
    b->sides.reserve(2 * n_tasks);
    frames.reserve(6 * n_tasks);
    partner.reserve(2 * n_tasks);
    for (uint64_t t = 0; t < n_tasks; ++t) {
        const sph_task& tk = tasks[t];
        b->task_side0[t] = (uint32_t)b->sides.size();
        if (tk.ci < 0 || (uint32_t)tk.ci >= n_cells || tk.cj < -1 || (tk.cj >= 0 && (uint32_t)tk.cj >= n_cells) || tk.cj == tk.ci)
            return fail(SPH_ERR_RANGE, "task %llu references cells (%d, %d); the store has %u", (unsigned long long)t, tk.ci, tk.cj, n_cells);
        for (int side = 0; side < (tk.cj >= 0 ? 2 : 1); ++side) {
            const uint32_t c = (uint32_t)(side == 0 ? tk.ci : tk.cj);
            const sph_cell& ce = store->cells[c];
            const uint32_t sidx = (uint32_t)b->sides.size();
            partner.push_back(tk.cj >= 0 ? (side == 0 ? sidx + 1 : sidx - 1) : sidx);
            b->sides.push_back(SideRec{(uint32_t)ce.first, ce.count, 0u, c});
            const double* fr = side == 0 ? tk.frame_i : tk.frame_j;
            frames.insert(frames.end(), fr, fr + 3);
            b->n_instances += ce.count;
            b->max_count = std::max(b->max_count, ce.count);
        }
        const uint64_t ni = store->cells[tk.ci].count;
        if (tk.cj >= 0) { ++b->n_pair; b->n_candidates += 2 * ni * store->cells[tk.cj].count; }
        else { ++b->n_self; b->n_candidates += ni * ni; }
    }
    b->task_side0[n_tasks] = (uint32_t)b->sides.size();
    b->n_sides = (uint32_t)b->sides.size();
    // a loop item carries its source count as nt_ns = targets | count << 7 (32 bits)
    if (b->max_count >= (1u << 25)) return fail(SPH_ERR_RANGE, "a cell of %u particles: the loops' item tables hold cell counts below 2^25", b->max_count);
    b->side_frames = frames;

    // per-cell occurrence lists in ascending (task, side) order = ascending side index
    std::vector<uint32_t> occ_count(n_cells, 0);
    for (const SideRec& s : b->sides) ++occ_count[s.cell];
    std::vector<uint32_t> occ_start(n_cells + 1, 0);
    for (uint32_t c = 0; c < n_cells; ++c) occ_start[c + 1] = occ_start[c] + occ_count[c];
    std::vector<uint32_t>& occ_side = b->occ_side;
    occ_side.resize(b->n_sides);
    std::vector<uint32_t> cur(occ_start.begin(), occ_start.end() - 1);
    for (uint32_t s = 0; s < b->n_sides; ++s) occ_side[cur[b->sides[s].cell]++] = s;
    std::vector<CellChunk> cell_chunks;
    b->cell_chunk0.assign(n_cells + 1, 0);
    for (uint32_t c = 0; c < n_cells; ++c) {
        b->cell_chunk0[c] = (uint32_t)cell_chunks.size();
        if (!occ_count[c]) continue;
        ++b->n_cells_touched;
        b->max_nocc = std::max(b->max_nocc, occ_count[c]);
        const sph_cell& ce = store->cells[c];
        for (uint32_t k = 0; k < ce.count; k += 32)
            cell_chunks.push_back(CellChunk{(uint32_t)ce.first + k, std::min(32u, ce.count - k), k, occ_start[c], occ_count[c]});
    }
    b->n_cell_chunks = (uint32_t)cell_chunks.size();
    b->cell_chunk0[n_cells] = b->n_cell_chunks;
    b->n_occ = b->n_sides;

    if (int32_t rc = upload(cell_chunks, &b->d_cell_chunks)) return rc;
    std::vector<double> occ_frames(3 * (size_t)b->n_sides);
    for (uint32_t o = 0; o < b->n_sides; ++o) std::copy_n(&frames[3 * (size_t)occ_side[o]], 3, &occ_frames[3 * (size_t)o]);
    if (int32_t rc = upload(occ_frames, &b->d_occ_frames)) return rc;
    for (uint32_t rec : {16u, 20u, 52u, 40u, 72u})
        if (int32_t rc = ensure_offsets(b, rec, nullptr)) return rc;

    // loop work items (one per 64-target chunk of a block) for the canonical record sizes of the two loops, cell-major: the
    // chunks of a cell's occurrences follow one another, so the warps that work on one cell run close together in time and
    // its blocks are still in L2
    {
        const std::vector<uint64_t> &o16 = b->offsets.at(16).h_off, &o20 = b->offsets.at(20).h_off, &o52 = b->offsets.at(52).h_off;
        const std::vector<uint64_t> &o40 = b->offsets.at(40).h_off, &o72 = b->offsets.at(72).h_off;
        std::vector<LoopItem> dens, forc, grad, forc3;
        std::vector<ItemSide>& ids = b->item_side;
        for (uint32_t c = 0; c < n_cells; ++c)
            for (uint32_t o = occ_start[c]; o < occ_start[c + 1]; ++o) {
                const uint32_t tgt = occ_side[o], src = partner[tgt];
                const uint32_t cnt = b->sides[tgt].count;
                for (uint32_t k = 0, kc = 0; k < cnt; k += kLoopTargets, ++kc) {
                    const uint32_t nt_ns = std::min(kLoopTargets, cnt - k) | b->sides[src].count << 7;
                    const uint32_t u = kLoopTargets / 32;                                // 32 records of r bytes = r units of 128 bytes
                    ids.push_back(ItemSide{tgt, src, kc});
                    dens.push_back(LoopItem{(uint32_t)(o20[tgt] / 128) + kc * 5 * u, (uint32_t)(o20[src] / 128), (uint32_t)(o16[tgt] / 128) + kc * 4 * u, nt_ns});
                    forc.push_back(LoopItem{(uint32_t)(o52[tgt] / 128) + kc * 13 * u, (uint32_t)(o52[src] / 128), (uint32_t)(o20[tgt] / 128) + kc * 5 * u, nt_ns});
                    grad.push_back(LoopItem{(uint32_t)(o40[tgt] / 128) + kc * 10 * u, (uint32_t)(o40[src] / 128), (uint32_t)(o16[tgt] / 128) + kc * 4 * u, nt_ns});
                    forc3.push_back(LoopItem{(uint32_t)(o72[tgt] / 128) + kc * 18 * u, (uint32_t)(o72[src] / 128), (uint32_t)(o20[tgt] / 128) + kc * 5 * u, nt_ns});
                }
            }
        // Longest first (occupancies of 5 .. 10^5 per cell).  Warps take items round-robin, so with
        // items in descending cost every warp gets a similar mix and the one 10^5 x 10^5 task starts at once instead of being
        // the tail.  Cost classes are powers of two of targets x sources and the sort is stable: inside a class the order stays
        // cell-major, and a batch whose items all cost the same (grids of equal cells) keeps its order.
        {
            auto cls = [](const LoopItem& it) { const uint64_t c = (uint64_t)(it.nt_ns & 127u) * (it.nt_ns >> 7); int k = 0; while ((c >> k) > 1) ++k; return k; };
            std::vector<uint32_t> order(dens.size());
            for (uint32_t i = 0; i < order.size(); ++i) order[i] = i;
            std::stable_sort(order.begin(), order.end(), [&](uint32_t x, uint32_t y) { return cls(dens[x]) > cls(dens[y]); });
            auto apply = [&](std::vector<LoopItem>& v) { std::vector<LoopItem> w(v.size()); for (size_t i = 0; i < v.size(); ++i) w[i] = v[order[i]]; v.swap(w); };
            apply(dens); apply(forc); apply(grad); apply(forc3);
            { std::vector<ItemSide> w(ids.size()); for (size_t i = 0; i < ids.size(); ++i) w[i] = ids[order[i]]; ids.swap(w); }
            uint64_t worst = 0;
            for (const LoopItem& it : dens) worst = std::max(worst, (uint64_t)(it.nt_ns & 127u) * (it.nt_ns >> 7));
            b->max_item_candidates = worst;
        }
        b->n_items = (uint32_t)dens.size();
        if (int32_t rc = upload(dens, &b->d_items_density)) return rc;
        if (int32_t rc = upload(forc, &b->d_items_force)) return rc;
        if (int32_t rc = upload(grad, &b->d_items_gradient)) return rc;
        if (int32_t rc = upload(forc3, &b->d_items_force3)) return rc;
    }

    *out = holder.release();
    return SPH_OK;
    SPH_API_END
}

int32_t sph_batch_destroy(sph_batch* b) {
    if (!b) return SPH_OK;
    cudaFree(b->d_cell_chunks); cudaFree(b->d_occ_frames); cudaFree(b->d_items_density); cudaFree(b->d_items_force); cudaFree(b->d_items_gradient); cudaFree(b->d_items_force3);
    for (auto& kv : b->offsets) { cudaFree(kv.second.d_off128); cudaFree(kv.second.d_occ_off128); }
    for (SlotTables& sl : b->slots) { cudaFree(sl.d_chunks); cudaFree(sl.d_slot_off128); cudaFree(sl.d_zero_frames); cudaFree(sl.d_items); cudaFree(sl.d_item_frames); }
    delete b;
    return SPH_OK;
}

int32_t sph_batch_get_info(const sph_batch* b, sph_batch_info* info) {
    if (!b || !info) return fail(SPH_ERR_INVALID_ARG, "NULL argument");
    info->n_tasks = b->n_tasks; info->n_self = b->n_self; info->n_pair = b->n_pair; info->n_sides = b->n_sides;
    info->n_instances = b->n_instances; info->n_candidates = b->n_candidates; info->n_cells_touched = b->n_cells_touched;
    info->n_segments = b->n_segments; info->max_count = b->max_count; info->n_items = b->n_items; info->max_item_candidates = b->max_item_candidates;
    return SPH_OK;
}

int32_t sph_batch_buffer_bytes(const sph_batch* b, const sph_attrset* set, uint64_t* bytes_out) {
    if (!b || !bytes_out) return fail(SPH_ERR_INVALID_ARG, "NULL argument");
    SPH_API_BEGIN
    uint32_t rec;
    if (int32_t rc = attrset_check(set, &rec)) return rc;
    const OffsetTable* ot;
    if (int32_t rc = ensure_offsets(b, rec, &ot)) return rc;
    *bytes_out = ot->total;
    return SPH_OK;
    SPH_API_END
}

int32_t sph_batch_block_offsets(const sph_batch* b, const sph_attrset* set, uint64_t* off_out, uint64_t* seg_off_out) {
    if (!b || !off_out) return fail(SPH_ERR_INVALID_ARG, "NULL argument");
    SPH_API_BEGIN
    uint32_t rec;
    if (int32_t rc = attrset_check(set, &rec)) return rc;
    const OffsetTable* ot;
    if (int32_t rc = ensure_offsets(b, rec, &ot)) return rc;
    for (uint64_t t = 0; t < b->n_tasks; ++t) {
        off_out[2 * t] = ot->h_off[b->task_side0[t]];
        off_out[2 * t + 1] = b->task_side0[t + 1] - b->task_side0[t] == 2 ? ot->h_off[b->task_side0[t] + 1] : UINT64_MAX;
    }
    if (seg_off_out) std::copy(ot->seg_off.begin(), ot->seg_off.end(), seg_off_out);
    return SPH_OK;
    SPH_API_END
}

}  // extern "C"
