// PACK and UNPACK kernels: pure data movement, HBM-bound.  Both are CELL-centric: a cell's particles
// are read (written) once per launch and copied to (reduced from) every block the cell occurs in.
//
// pack (pack_kernel): one warp per 32-particle chunk of a cell and a slice of the cell's occurrences.  The chunk's structs
//   are staged once into shared memory with coalesced cp.async (only the 16-byte pieces that hold requested fields), re-sliced
//   once into the compact record stream (a "template"), and per occurrence the three x words are patched with
//   f32(x - frame) and ONE bulk copy (cp.async.bulk shared -> global) writes the block's slice.  See the kernel's comments.
//
// unpack (unpack_kernel): one warp per 32-particle chunk of a cell, a two-stage pipeline of rounds: the chunk's slice of
//   every block of the round is fetched by one bulk copy per slice (global -> shared, mbarrier), then one lane per particle
//   applies the per-field operator (+=, max, =) over the slices in ascending (task, side) order in f32: bit-reproducible, no
//   atomics, no races (a particle is owned by exactly one warp per launch); the store's fields are read and written once.
#include <algorithm>

#include "internal.h"
#include "ptx.cuh"

namespace sph {

namespace {

using namespace ptx;

#ifndef SPH_PACK_WARPS
#define SPH_PACK_WARPS 4
#endif
#ifndef SPH_PACK_K
#define SPH_PACK_K 4
#endif
#ifndef SPH_UNPACK_WARPS
#define SPH_UNPACK_WARPS 2
#endif
constexpr int kPackWarps = SPH_PACK_WARPS;
constexpr int kUnpackWarps = SPH_UNPACK_WARPS;

constexpr int kPackK = SPH_PACK_K;                      // record-stream templates per set; two sets alternate
constexpr uint32_t kPackTableOcc = 32;         // occurrences whose block offsets and frames are staged at a time
constexpr uint32_t kPackTableBytes = kPackTableOcc * (4 + 24);

template <int NIT>
__global__ void __launch_bounds__(kPackWarps * 32)
pack_kernel(Program prog, const CellChunk* __restrict__ cell_chunks, const uint32_t* __restrict__ occ_off128,
            const double* __restrict__ occ_frames, uint32_t n_cell_chunks, uint32_t slices, char* __restrict__ buf) {
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t R = prog.rec_words;
    const uint32_t templ_bytes = 128 * R;                           // 32 records
    unsigned char* stage = smem + (size_t)warp * (prog.smem_per_warp + 2 * kPackK * templ_bytes + 2 * kPackTableBytes);
    unsigned char* templ = stage + prog.smem_per_warp;              // 2 sets of kPackK copies
    unsigned char* tables = templ + 2 * kPackK * templ_bytes;       // 2 x { double frames[32][3]; uint32_t off128[32]; }

    // which staging word feeds output word g = 4 (lane + 32 it) + j of a chunk's record stream
    uint32_t src[NIT][4];
#pragma unroll
    for (int it = 0; it < NIT; ++it)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t g = 4 * (lane + 32 * it) + j;
            const uint32_t k = g / R, w = g - k * R;
            src[it][j] = k < 32 ? prog.word[w].a + k * prog.word[w].stride : 0;
        }
    const uint32_t xw0 = prog.xw[0], xw1 = prog.xw[1], xw2 = prog.xw[2];
    const bool xrel = prog.xrel != 0;

    // item -> its cell chunk and its slice [ob, oe) of the cell's occurrences (empty for a short cell)
    const uint32_t n_items = n_cell_chunks * slices, item_step = gridDim.x * kPackWarps;
    auto item_range = [&](uint32_t it, CellChunk* c, uint32_t* o_b, uint32_t* o_e) {
        const uint32_t cc = it / slices, sl = it - cc * slices;
        *c = cell_chunks[cc];
        const uint32_t per = (c->nocc + slices - 1) / slices;
        *o_b = min(c->nocc, sl * per); *o_e = min(c->nocc, *o_b + per);
    };
    // block offsets and frames of occurrences [o0, o0 + cnt) of a cell -> table t (asynchronous)
    auto stage_table = [&](const CellChunk& c, uint32_t o0, uint32_t cnt, uint32_t t) {
        unsigned char* tb = tables + t * kPackTableBytes;
        if (lane < cnt) {
            cp_async<4>(tb + 24 * kPackTableOcc + 4 * lane, occ_off128 + c.occ0 + o0 + lane);
            if (xrel) {
                const double* f = occ_frames + 3 * (size_t)(c.occ0 + o0 + lane);
                cp_async<8>(tb + 24 * lane, f); cp_async<8>(tb + 24 * lane + 8, f + 1); cp_async<8>(tb + 24 * lane + 16, f + 2);
            }
        }
    };
    // the chunk's structs -> the staging area (asynchronous)
    auto stage_chunk = [&](const CellChunk& c) {
        for (uint32_t u = 0; u < prog.n_sub_used; ++u) {
            const PackSub su = prog.su[u];
            const char* g = su.base + (uint64_t)c.first * su.stride;
            unsigned char* dst = stage + su.smem_base;
            const uint32_t nbytes = c.count * su.stride;
            if (su.gran == 16) {
                const uint32_t nvec = nbytes >> 4;
                if (su.mask == 0xFFFFFFFFu) {
                    for (uint32_t v = lane; v < nvec; v += 32) cp_async<16>(dst + 16 * v, g + 16 * v);
                } else {
                    const uint32_t per16 = su.stride >> 4;
                    for (uint32_t v = lane; v < nvec; v += 32)
                        if (su.mask >> (v & (per16 - 1)) & 1) cp_async<16>(dst + 16 * v, g + 16 * v);
                }
            } else if (su.gran == 8) {
                for (uint32_t v = lane; v < (nbytes >> 3); v += 32) cp_async<8>(dst + 8 * v, g + 8 * v);
            } else {
                for (uint32_t v = lane; v < (nbytes >> 2); v += 32) cp_async<4>(dst + 4 * v, g + 4 * v);
            }
        }
    };

    uint32_t item = blockIdx.x * kPackWarps + warp;
    if (item >= n_items) return;
    CellChunk ch, ch_next{};
    uint32_t ob, oe, ob_next = 0, oe_next = 0, tcur = 0;
    item_range(item, &ch, &ob, &oe);
    if (ob < oe) { stage_chunk(ch); stage_table(ch, ob, min(kPackTableOcc, oe - ob), 0); }

    for (; item < n_items; item += item_step, tcur ^= 1) {
        const bool has_next = item + item_step < n_items;
        if (has_next) item_range(item + item_step, &ch_next, &ob_next, &oe_next);     // in flight during the template build
        cp_async_wait_all();
        __syncwarp();
        const uint32_t n = ch.count;
        const bool live = ob < oe && lane < n;
        // (1) one lane per particle: keep x in registers (it is re-based for every occurrence); widen time_bin
        double x0 = 0., x1 = 0., x2 = 0.;
        if (xrel && live) {
            const unsigned char* px = stage + prog.x_src + lane * prog.x_stride;
            x0 = *reinterpret_cast<const double*>(px); x1 = *reinterpret_cast<const double*>(px + 8); x2 = *reinterpret_cast<const double*>(px + 16);
        }
        if (prog.tb && live)
            *reinterpret_cast<uint32_t*>(stage + prog.tb_dst + 4 * lane) = stage[prog.tb_src + lane * prog.tb_stride];
        if (lane < kPackK) bulk_wait_read<0>();       // the previous item's bulk stores have read the templates
        __syncwarp();

        // (2) re-slice the staging area into the record stream, every template copy; the x words are patched per occurrence
        if (ob < oe) {
#pragma unroll
            for (int it = 0; it < NIT; ++it) {
                const uint32_t v = lane + 32 * it;
                if (v < 8 * R) {
                    uint4 o;
                    o.x = *reinterpret_cast<const uint32_t*>(stage + src[it][0]);
                    o.y = *reinterpret_cast<const uint32_t*>(stage + src[it][1]);
                    o.z = *reinterpret_cast<const uint32_t*>(stage + src[it][2]);
                    o.w = *reinterpret_cast<const uint32_t*>(stage + src[it][3]);
#pragma unroll
                    for (int c = 0; c < 2 * kPackK; ++c) *reinterpret_cast<uint4*>(templ + c * templ_bytes + 16 * v) = o;
                }
            }
        }
        __syncwarp();   // the staging area is free: the next item's structs and table travel during this item's copies
        if (has_next && ob_next < oe_next) { stage_chunk(ch_next); stage_table(ch_next, ob_next, min(kPackTableOcc, oe_next - ob_next), tcur ^ 1); }

        // (3) one bulk copy (TMA) of a template per occurrence of the cell (task side), x re-based to that side's frame.
        //     Occurrences go in groups of kPackK; the two template sets alternate, so a group is patched while the previous
        //     group's copies are still reading the other set.
        const uint32_t bytes = (n * R * 4 + 15) & ~15u;      // a last partial vector spills into the block's pad bytes
        const uint64_t chunk_off = (uint64_t)ch.k0 * R * 4;
        unsigned char* tb = tables + tcur * kPackTableBytes;
        uint32_t t0 = ob;                                    // first occurrence the table holds
        for (uint32_t o = ob, g = 0; o < oe; o += kPackK, ++g) {
            if (o + kPackK > t0 + kPackTableOcc && t0 + kPackTableOcc < oe) {     // a cell with many occurrences: refill the table
                __syncwarp();
                t0 = o;
                if (lane < min(kPackTableOcc, oe - t0)) {
                    reinterpret_cast<uint32_t*>(tb + 24 * kPackTableOcc)[lane] = __ldg(occ_off128 + ch.occ0 + t0 + lane);
                    const double* f = occ_frames + 3 * (size_t)(ch.occ0 + t0 + lane);
                    double* d = reinterpret_cast<double*>(tb + 24 * lane);
                    if (xrel) { d[0] = __ldg(f); d[1] = __ldg(f + 1); d[2] = __ldg(f + 2); }
                }
            }
            unsigned char* set = templ + (g & 1) * kPackK * templ_bytes;
            if (g >= 2 && lane < kPackK) bulk_wait_read<1>();     // the group before last has read this set
            __syncwarp();
            if (xrel && live) {
#pragma unroll
                for (int k = 0; k < kPackK; ++k) {
                    if (o + k < oe) {
                        const double* f = reinterpret_cast<const double*>(tb + 24 * (o + k - t0));
                        float* rec = reinterpret_cast<float*>(set + k * templ_bytes) + lane * R;
                        if (xw0 != 0xFFFFFFFFu) rec[xw0] = __double2float_rn(__dsub_rn(x0, f[0]));
                        if (xw1 != 0xFFFFFFFFu) rec[xw1] = __double2float_rn(__dsub_rn(x1, f[1]));
                        if (xw2 != 0xFFFFFFFFu) rec[xw2] = __double2float_rn(__dsub_rn(x2, f[2]));
                    }
                }
            }
            fence_proxy_async();      // template words written through the generic proxy are read by the bulk copy
            __syncwarp();
            if (lane < kPackK) {
                if (o + lane < oe) {
                    const uint32_t o128 = reinterpret_cast<const uint32_t*>(tb + 24 * kPackTableOcc)[o + lane - t0];
                    bulk_s2g(buf + (uint64_t)o128 * 128 + chunk_off, set + lane * templ_bytes, bytes);
                }
                bulk_commit();
            }
        }
        ch = ch_next; ob = ob_next; oe = oe_next;
    }
    if (lane < kPackK) bulk_wait_read<0>();    // shared memory must outlive the copies that read it
}

// ---------------------------------------------------------------------------------------------------------

// One warp per 32-particle chunk of a cell, as a two-stage pipeline of ROUNDS (a round = up to `slots` of the blocks the
// cell occurs in, normally all of them):
//  (1) fetch: the chunk's slice of every block of the round travels global -> shared memory as ONE bulk copy (TMA,
//      cp.async.bulk) per slice, each issued by its own lane and all completing on the ring's mbarrier: a whole round is
//      one instruction per lane, holds no registers while in flight, and the NEXT round (of this chunk, or the first of
//      the warp's next chunk) is issued into the other ring before the current one is waited for; rings are small (9
//      slices, ~5 KB) so that 18 warps share an SM: one warp's reduction overlaps the other warps' fetches;
//  (2) reduce: one lane per particle walks the slices in ascending (task, side) order.  With the lane owning a
//      record, the operator of word j (+=, max, =) is the same in every lane: no per-lane dispatch, no divergence.
//      Records are read with VEC-word shared loads (stride = record length: conflict-free when R / VEC is odd).
//  Words are processed in groups of GW; a record longer than GW keeps its running values in a scratch slot.
// The store's own values of the next chunk (the starting point of its sums) are loaded one round ahead as well.
template <int VEC, int GW>
__global__ void __launch_bounds__(kUnpackWarps * 32)
unpack_kernel(StoreView view, Program prog, const CellChunk* __restrict__ cell_chunks, const uint32_t* __restrict__ occ_off128,
              uint32_t n_cell_chunks, const char* __restrict__ buf, uint32_t slots, uint32_t last_only, uint32_t all_sum, uint32_t from_zero) {
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t R = prog.rec_words;
    const uint32_t slot_bytes = 128 * R;
    const bool single = R <= GW;                       // the whole record lives in registers; else one slot of scratch
    const uint32_t ring_bytes = slots * slot_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem) + 2 * warp;       // one mbarrier per ring
    unsigned char* wbase = smem + 128 + (size_t)warp * (2 * ring_bytes + (single ? 0u : slot_bytes));
    float* scratch = reinterpret_cast<float*>(wbase + 2 * ring_bytes);   // [R][32]

    const uint32_t cc_step = gridDim.x * kUnpackWarps;
    const uint32_t cc0 = blockIdx.x * kUnpackWarps + warp;
    if (cc0 >= n_cell_chunks) return;
    if (lane == 0) { mbar_init(bars, 1); mbar_init(bars + 1, 1); fence_mbar_init(); }
    __syncwarp();

    // store access of word w of particle p
    auto word_addr = [&](uint32_t w, uint64_t p) { return view.base[prog.word[w].sub] + p * prog.word[w].stride + prog.word[w].a; };
    auto is_reduced = [&](uint32_t w) { return prog.word[w].kind == W_SUM || prog.word[w].kind == W_MAX; };

    // the running values of a chunk start from the store's own (reduced words only)
    auto load_own = [&](float (&a)[GW], const CellChunk& c) {
#pragma unroll
        for (int j = 0; j < GW; ++j) a[j] = 0.f;
        if (!single || from_zero || lane >= c.count) return;
        const uint64_t p = (uint64_t)c.first + lane;
#pragma unroll
        for (int j = 0; j < GW; ++j) {
            if ((uint32_t)j >= R) continue;
            if (j % 4 == 0 && j + 3 < GW && prog.vec4[j]) {
                const float4 t = *reinterpret_cast<const float4*>(word_addr(j, p));
                a[j] = t.x; if (j + 1 < GW) a[j + 1] = t.y; if (j + 2 < GW) a[j + 2] = t.z; if (j + 3 < GW) a[j + 3] = t.w;
            } else if (!(prog.vec4[4 * (j / 4)] && 4 * (j / 4) + 3 < GW) && is_reduced(j)) {
                a[j] = *reinterpret_cast<const float*>(word_addr(j, p));
            }
        }
    };

    // a cursor over the rounds of the warp's chunks
    struct Cur { CellChunk ch; uint32_t cc, ob, per_round; };
    auto enter = [&](Cur& c, uint32_t cc, const CellChunk& ch) {
        c.cc = cc; c.ch = ch;
        c.ob = last_only ? ch.nocc - 1 : 0;
        const uint32_t n_o = ch.nocc - c.ob, n_rounds = (n_o + slots - 1) / slots;
        c.per_round = (n_o + n_rounds - 1) / n_rounds;                    // <= slots <= 32
    };
    // one round into ring r: lane u fetches the chunk's slice of block (ob + u)
    auto issue = [&](const Cur& c, uint32_t r) {
        const uint32_t lim = min(c.per_round, c.ch.nocc - c.ob);
        const uint32_t bytes = (c.ch.count * R * 4 + 15) & ~15u;          // a last partial vector reads into the block's pad bytes
        const uint32_t tbl = lane < lim ? __ldg(occ_off128 + c.ch.occ0 + c.ob + lane) : 0u;
        if (lane == 0) mbar_expect_tx(bars + r, lim * bytes);
        __syncwarp();
        if (lane < lim) bulk_g2s(wbase + r * ring_bytes + lane * slot_bytes, buf + (uint64_t)tbl * 128 + (uint64_t)c.ch.k0 * R * 4, bytes, bars + r);
    };

    // one group of words [g0, g0 + nw) reduced over the `lim` slices of a ring, in slice order
    auto reduce_group = [&](float (&acc)[GW], const unsigned char* ring, uint32_t g0, uint32_t nw, uint32_t lim) {
        const unsigned char* rec = ring + (lane * R + g0) * 4;
        if constexpr (VEC == 1) {
            // odd record length: scalar shared loads are conflict-free, so every word runs its own loop over the slices with its
            // operator hoisted out of it (warp-uniform): one load and one operation per slice and word, loads batched ahead
            if (!all_sum) {
#pragma unroll
                for (int j = 0; j < GW; ++j) {
                    if ((uint32_t)j >= nw) continue;
                    const uint32_t kind = prog.word[g0 + j].kind;
                    const unsigned char* rj = rec + 4 * j;
                    if (kind == W_SUM) {
#pragma unroll 9
                        for (uint32_t u = 0; u < lim; ++u) acc[j] = __fadd_rn(acc[j], *reinterpret_cast<const float*>(rj + u * slot_bytes));
                    } else if (kind == W_MAX) {
#pragma unroll 9
                        for (uint32_t u = 0; u < lim; ++u) acc[j] = fmaxf(acc[j], *reinterpret_cast<const float*>(rj + u * slot_bytes));
                    } else {
                        acc[j] = *reinterpret_cast<const float*>(rj + (lim - 1) * slot_bytes);      // overwrite: the last slice wins
                    }
                }
                return;
            }
        }
        uint32_t m_sum[GW], m_red[GW];
#pragma unroll
        for (int j = 0; j < GW; ++j) {
            const uint32_t kind = (uint32_t)j < nw ? prog.word[g0 + j].kind : (uint32_t)W_SKIP;
            m_sum[j] = kind == W_SUM ? 0xFFFFFFFFu : 0u;
            m_red[j] = kind == W_SUM || kind == W_MAX ? 0xFFFFFFFFu : 0u;
        }
#pragma unroll 4
        for (uint32_t u = 0; u < lim; ++u, rec += slot_bytes) {
            float rv[GW];
#pragma unroll
            for (int j = 0; j < GW; j += VEC) {
                if ((uint32_t)j >= nw) { for (int q = 0; q < VEC; ++q) rv[j + q] = 0.f; continue; }
                if constexpr (VEC == 4) {
                    const float4 t = *reinterpret_cast<const float4*>(rec + 4 * j);
                    rv[j] = t.x; rv[j + 1] = t.y; rv[j + 2] = t.z; rv[j + 3] = t.w;
                } else if constexpr (VEC == 2) {
                    const float2 t = *reinterpret_cast<const float2*>(rec + 4 * j);
                    rv[j] = t.x; rv[j + 1] = t.y;
                } else {
                    rv[j] = *reinterpret_cast<const float*>(rec + 4 * j);
                }
            }
            if (all_sum) {
#pragma unroll
                for (int j = 0; j < GW; ++j) acc[j] = __fadd_rn(acc[j], rv[j]);
            } else {
#pragma unroll
                for (int j = 0; j < GW; ++j) {   // bit-select, not a branch: sum where m_sum, max where m_red only, else the record's value
                    const uint32_t s = __float_as_uint(__fadd_rn(acc[j], rv[j])), m = __float_as_uint(fmaxf(acc[j], rv[j]));
                    const uint32_t t = (s & m_sum[j]) | (m & ~m_sum[j]);
                    acc[j] = __uint_as_float((t & m_red[j]) | (__float_as_uint(rv[j]) & ~m_red[j]));
                }
            }
        }
    };

    Cur F;                                   // the round being fetched; the consumer follows one round behind
    enter(F, cc0, cell_chunks[cc0]);
    CellChunk ch_pre{};                      // descriptor of the warp's next chunk, loaded a chunk ahead
    if (cc0 + cc_step < n_cell_chunks) ch_pre = cell_chunks[cc0 + cc_step];
    float acc[GW], acc_pre[GW];
    load_own(acc_pre, F.ch);
    issue(F, 0);
    bool f_valid = true;
    for (uint32_t it = 0; f_valid; ++it) {
        const Cur C = F;
        const bool c_first = C.ob == (last_only ? C.ch.nocc - 1 : 0u);
        const uint32_t lim = min(C.per_round, C.ch.nocc - C.ob);
        const bool c_last = C.ob + lim >= C.ch.nocc;
        if (c_first) {
#pragma unroll
            for (int j = 0; j < GW; ++j) acc[j] = acc_pre[j];
        }
        // advance the fetch cursor and put its round in flight (the other ring was released at the end of the previous iteration)
        F.ob += F.per_round;
        if (F.ob >= F.ch.nocc) {
            const uint32_t cc = F.cc + cc_step;
            f_valid = cc < n_cell_chunks;
            if (f_valid) {
                enter(F, cc, ch_pre);
                if (cc + cc_step < n_cell_chunks) ch_pre = cell_chunks[cc + cc_step];
                load_own(acc_pre, F.ch);
            }
        }
        if (f_valid) issue(F, (it + 1) & 1);

        const unsigned char* ring = wbase + (it & 1) * ring_bytes;
        const bool live = lane < C.ch.count;
        const uint64_t p = (uint64_t)C.ch.first + lane;
        if (!single && c_first)
            for (uint32_t w = 0; w < R; ++w)
                scratch[w * 32 + lane] = live && !from_zero && is_reduced(w) ? *reinterpret_cast<const float*>(word_addr(w, p)) : 0.f;
        mbar_wait(bars + (it & 1), (it >> 1) & 1);
        if (single) {
            reduce_group(acc, ring, 0, R, lim);
        } else {
            for (uint32_t g0 = 0; g0 < R; g0 += GW) {
                const uint32_t nw = min((uint32_t)GW, R - g0);
                float a2[GW];
#pragma unroll
                for (int j = 0; j < GW; ++j) a2[j] = (uint32_t)j < nw ? scratch[(g0 + j) * 32 + lane] : 0.f;
                reduce_group(a2, ring, g0, nw, lim);
#pragma unroll
                for (int j = 0; j < GW; ++j) if ((uint32_t)j < nw) scratch[(g0 + j) * 32 + lane] = a2[j];
            }
        }
        if (c_last && live) {
            if (single) {
#pragma unroll
                for (int j = 0; j < GW; ++j) {
                    if ((uint32_t)j >= R) continue;
                    const int j4 = 4 * (j / 4);
                    if (j4 + 3 < GW && prog.vec4[j4]) {
                        if (j == j4) *reinterpret_cast<float4*>(word_addr(j, p)) = make_float4(acc[j4], acc[j4 + 1 < GW ? j4 + 1 : j4], acc[j4 + 2 < GW ? j4 + 2 : j4], acc[j4 + 3 < GW ? j4 + 3 : j4]);
                    } else if (prog.word[j].kind == W_ASSIGN_BYTE) {
                        *reinterpret_cast<unsigned char*>(word_addr(j, p)) = (unsigned char)__float_as_uint(acc[j]);
                    } else {
                        *reinterpret_cast<float*>(word_addr(j, p)) = acc[j];
                    }
                }
            } else {
                for (uint32_t w = 0; w < R; ++w) {
                    const float v = scratch[w * 32 + lane];
                    if (prog.word[w].kind == W_ASSIGN_BYTE) *reinterpret_cast<unsigned char*>(word_addr(w, p)) = (unsigned char)__float_as_uint(v);
                    else *reinterpret_cast<float*>(word_addr(w, p)) = v;
                }
            }
        }
        fence_proxy_async();          // this ring's generic-proxy reads are ordered before the bulk copy that refills it
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------------------

// ------------------------------------------------------------------------------------------------- pack passes (loop fission)
//
// GPU analogue of the paper's split pack loops (by-struct, by-element, by-type, by-struct-and-type): ONE pass
// writes a subset of the record words -- each selected word is read once per particle straight from its substruct array and
// stored into its place in the record of every block the cell occurs in.  The passes of a partition together write exactly
// what the fused pack_kernel writes; every pass re-touches every output sector, which is what the comparison measures.
__global__ void __launch_bounds__(128)
pack_pass_kernel(StoreView view, PassProgram pp, const CellChunk* __restrict__ cell_chunks, const uint32_t* __restrict__ occ_off128,
                 const double* __restrict__ occ_frames, uint32_t n_cell_chunks, char* __restrict__ buf) {
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t rec_bytes = 4 * pp.rec_words;
    for (uint32_t cc = blockIdx.x * 4 + (threadIdx.x >> 5); cc < n_cell_chunks; cc += gridDim.x * 4) {
        const CellChunk c = cell_chunks[cc];
        if (lane >= c.count) continue;
        const uint64_t p = (uint64_t)c.first + lane;
        const uint64_t rec0 = (uint64_t)(c.k0 + lane) * rec_bytes;
        for (uint32_t s = 0; s < pp.n_sel; ++s) {
            const PassWord w = pp.sel[s];
            const char* src = view.base[w.sub] + p * w.stride + w.off;
            if (w.kind == W_XREL) {
                const double x = *reinterpret_cast<const double*>(src);
                for (uint32_t o = 0; o < c.nocc; ++o)
                    *reinterpret_cast<float*>(buf + (uint64_t)occ_off128[c.occ0 + o] * 128 + rec0 + 4 * w.w) = (float)(x - occ_frames[3 * (size_t)(c.occ0 + o) + w.comp]);
            } else {
                const uint32_t v = w.kind == W_TIMEBIN ? (uint32_t) * reinterpret_cast<const unsigned char*>(src) : *reinterpret_cast<const uint32_t*>(src);
                for (uint32_t o = 0; o < c.nocc; ++o)
                    *reinterpret_cast<uint32_t*>(buf + (uint64_t)occ_off128[c.occ0 + o] * 128 + rec0 + 4 * w.w) = v;
            }
        }
    }
}

__global__ void zero_kernel(StoreView view, Program prog, uint64_t n) {
    const uint64_t total = n * prog.rec_words;
    for (uint64_t g = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; g < total; g += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t p = g / prog.rec_words;
        const WordDesc wd = prog.word[g - p * prog.rec_words];
        *reinterpret_cast<float*>(view.base[wd.sub] + p * wd.stride + wd.a) = 0.f;
    }
}

struct GhostLoc { uint32_t sub_rho, off_rho, sub_u, off_u, sub_p, off_p, sub_cs, off_cs; };

// f64 on purpose: N particles once per step, and it makes P, c_s the correctly rounded values of the formula
__global__ void ghost_kernel(StoreView view, GhostLoc loc, uint64_t n, double gamma) {
    const double gm1 = gamma - 1.0, g_gm1 = __dmul_rn(gamma, gm1);
    for (uint64_t p = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; p < n; p += (uint64_t)gridDim.x * blockDim.x) {
        const double rho = *reinterpret_cast<const float*>(view.base[loc.sub_rho] + p * view.stride[loc.sub_rho] + loc.off_rho);
        const double u = *reinterpret_cast<const float*>(view.base[loc.sub_u] + p * view.stride[loc.sub_u] + loc.off_u);
        *reinterpret_cast<float*>(view.base[loc.sub_p] + p * view.stride[loc.sub_p] + loc.off_p) = __double2float_rn(__dmul_rn(__dmul_rn(gm1, rho), u));
        *reinterpret_cast<float*>(view.base[loc.sub_cs] + p * view.stride[loc.sub_cs] + loc.off_cs) = __double2float_rn(__dsqrt_rn(__dmul_rn(g_gm1, u)));
    }
}

int32_t sm_count(int* out) { return device_sms(out); }

}  // namespace

// SM count of the current device, asked for on every launch (no process-wide cache: a process may use several devices)
int32_t device_sms(int* sms_out) {
    int dev = 0;
    SPH_CUDA_TRY(cudaGetDevice(&dev));
    SPH_CUDA_TRY(cudaDeviceGetAttribute(sms_out, cudaDevAttrMultiProcessorCount, dev));
    return SPH_OK;
}

namespace {

template <int NIT>
int32_t launch_pack_nit(const CellChunk* d_chunks, const double* d_occ_frames, const Program& prog, const uint32_t* d_occ_off128, char* d_buf, size_t smem, int sms,
                        uint32_t ncc, cudaStream_t st) {
    if (smem > 48 * 1024) SPH_CUDA_TRY(cudaFuncSetAttribute(pack_kernel<NIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // resident CTAs per SM (shared memory and 64 warps bound it); a cell's occurrences are split into `slices` items
    // when there are fewer cell chunks than about two rounds of resident warps
    const uint32_t per_sm = (uint32_t)std::max<size_t>(1, std::min<size_t>(64 / kPackWarps, (220 * 1024) / (smem + 1024)));
    const uint32_t resident_warps = (uint32_t)sms * per_sm * kPackWarps;
    const uint32_t slices = std::min(8u, std::max(1u, (2 * resident_warps + ncc - 1) / ncc));
    const uint64_t items = (uint64_t)ncc * slices;
    const uint32_t grid = (uint32_t)std::min<uint64_t>((items + kPackWarps - 1) / kPackWarps, (uint64_t)sms * per_sm);
    pack_kernel<NIT><<<grid, kPackWarps * 32, smem, st>>>(prog, d_chunks, d_occ_off128, d_occ_frames, ncc, slices, d_buf);
    return SPH_OK;
}

#ifndef SPH_UNPACK_MAXCTA
#define SPH_UNPACK_MAXCTA 16
#endif
#ifndef SPH_UNPACK_RING
#define SPH_UNPACK_RING 5760
#endif
// per ring: 9 slices of 32 x 20-byte records -- a cell of a periodic grid (27 blocks) takes three rounds; small rings let
// 9 CTAs (18 warps) share an SM, which is what overlaps one warp's reduction with the others' fetches (measured on
// configs[2]: 27-slice rings 0.36 ms, 9-slice rings 0.23 ms)
constexpr uint32_t kUnpackRingBytes = SPH_UNPACK_RING;

template <int VEC, int GW>
int32_t launch_unpack_t(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_occ_off128, const char* d_buf,
                        bool last_only, bool all_sum, bool from_zero, int sms, uint32_t cc0, uint32_t ncc, cudaStream_t st) {
    const uint32_t slot_bytes = 128 * prog.rec_words;
    const uint32_t extra = prog.rec_words <= (uint32_t)GW ? 0 : 1;      // scratch slot of a long record
    const uint32_t slots = last_only ? 1u : std::max(1u, std::min(std::min(32u, b->max_nocc), kUnpackRingBytes / slot_bytes));
    const size_t smem = 128 + (size_t)kUnpackWarps * (2 * slots + extra) * slot_bytes;      // mbarriers, then two rings (+ scratch) per warp
    if (smem > 48 * 1024) SPH_CUDA_TRY(cudaFuncSetAttribute(unpack_kernel<VEC, GW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const uint32_t per_sm = (uint32_t)std::max<size_t>(1, std::min<size_t>(SPH_UNPACK_MAXCTA, (227 * 1024) / (smem + 1024)));
    const uint32_t want = (ncc + kUnpackWarps - 1) / kUnpackWarps;
    const uint32_t grid = std::min(want, (uint32_t)sms * per_sm);
    unpack_kernel<VEC, GW><<<grid, kUnpackWarps * 32, smem, st>>>(view, prog, b->d_cell_chunks + cc0, d_occ_off128, ncc, d_buf, slots,
                                                                   last_only ? 1u : 0u, all_sum ? 1u : 0u, from_zero ? 1u : 0u);
    return SPH_OK;
}

}  // namespace

int32_t launch_pack_tables(const StoreView& view, const Program& prog_in, const CellChunk* d_chunks, const uint32_t* d_occ_off128, const double* d_occ_frames,
                           char* d_buf, uint32_t ncc, cudaStream_t st) {
    if (ncc == 0) return SPH_OK;
    Program prog = prog_in;
    for (uint32_t u = 0; u < prog.n_sub_used; ++u) prog.su[u].base = view.base[prog.su[u].sub];
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    const size_t smem = ((size_t)prog.smem_per_warp + 2 * kPackK * 128 * (size_t)prog.rec_words + 2 * kPackTableBytes) * kPackWarps;
    if (smem > 200 * 1024) return fail(SPH_ERR_UNSUPPORTED, "layout needs %zu bytes of staging per CTA", smem);
    const uint32_t nit = (prog.rec_words + 3) / 4;   // 16-byte vectors per lane for a full chunk: ceil(32 R / 4 / 32)
    int32_t rc;
    if (nit <= 1) rc = launch_pack_nit<1>(d_chunks, d_occ_frames, prog, d_occ_off128, d_buf, smem, sms, ncc, st);
    else if (nit <= 2) rc = launch_pack_nit<2>(d_chunks, d_occ_frames, prog, d_occ_off128, d_buf, smem, sms, ncc, st);
    else if (nit <= 4) rc = launch_pack_nit<4>(d_chunks, d_occ_frames, prog, d_occ_off128, d_buf, smem, sms, ncc, st);
    else if (nit <= 6) rc = launch_pack_nit<6>(d_chunks, d_occ_frames, prog, d_occ_off128, d_buf, smem, sms, ncc, st);
    else if (nit <= 9) rc = launch_pack_nit<9>(d_chunks, d_occ_frames, prog, d_occ_off128, d_buf, smem, sms, ncc, st);
    else rc = launch_pack_nit<12>(d_chunks, d_occ_frames, prog, d_occ_off128, d_buf, smem, sms, ncc, st);
    if (rc) return rc;
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_pack(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_occ_off128, char* d_buf,
                    uint32_t cc0, uint32_t ncc, cudaStream_t st) {
    return launch_pack_tables(view, prog, b->d_cell_chunks + cc0, d_occ_off128, b->d_occ_frames, d_buf, ncc, st);
}

int32_t launch_unpack(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_occ_off128, const char* d_buf,
                      bool last_only, bool from_zero, uint32_t cc0, uint32_t ncc, cudaStream_t st) {
    if (ncc == 0) return SPH_OK;
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    bool all_sum = true;
    for (uint32_t w = 0; w < prog.rec_words; ++w) all_sum &= prog.word[w].kind == W_SUM;
    const uint32_t R = prog.rec_words;
    int32_t rc;
    if (R % 4 == 0) rc = R % 8 == 0 ? launch_unpack_t<4, 8>(view, b, prog, d_occ_off128, d_buf, last_only, all_sum, from_zero, sms, cc0, ncc, st)
                                    : launch_unpack_t<4, 4>(view, b, prog, d_occ_off128, d_buf, last_only, all_sum, from_zero, sms, cc0, ncc, st);
    else if (R % 2 == 0) rc = launch_unpack_t<2, 8>(view, b, prog, d_occ_off128, d_buf, last_only, all_sum, from_zero, sms, cc0, ncc, st);
    else if (R % 5 == 0) rc = launch_unpack_t<1, 5>(view, b, prog, d_occ_off128, d_buf, last_only, all_sum, from_zero, sms, cc0, ncc, st);
    else rc = launch_unpack_t<1, 8>(view, b, prog, d_occ_off128, d_buf, last_only, all_sum, from_zero, sms, cc0, ncc, st);
    if (rc) return rc;
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_pack_pass(const StoreView& view, const PassProgram& pp, const CellChunk* d_chunks, const uint32_t* d_occ_off128, const double* d_occ_frames,
                         char* d_buf, uint32_t ncc, cudaStream_t st) {
    if (ncc == 0 || pp.n_sel == 0) return SPH_OK;
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    const uint32_t grid = std::min((ncc + 3) / 4, (uint32_t)sms * 16);
    pack_pass_kernel<<<grid, 128, 0, st>>>(view, pp, d_chunks, d_occ_off128, d_occ_frames, ncc, d_buf);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_zero(const StoreView& view, uint64_t n, const Program& prog, cudaStream_t st) {
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    const uint64_t total = n * prog.rec_words;
    const uint32_t grid = (uint32_t)std::min<uint64_t>((total + 255) / 256, (uint64_t)sms * 16);
    zero_kernel<<<grid, 256, 0, st>>>(view, prog, n);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_ghost(const StoreView& view, uint64_t n, const sph_layout& l, const sph_params& prm, cudaStream_t st) {
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    GhostLoc loc{l.loc[SPH_RHO].sub, l.loc[SPH_RHO].off, l.loc[SPH_U].sub, l.loc[SPH_U].off,
                 l.loc[SPH_P].sub, l.loc[SPH_P].off, l.loc[SPH_CS].sub, l.loc[SPH_CS].off};
    const uint32_t grid = (uint32_t)std::min<uint64_t>((n + 255) / 256, (uint64_t)sms * 16);
    ghost_kernel<<<grid, 256, 0, st>>>(view, loc, n, (double)prm.gamma);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
