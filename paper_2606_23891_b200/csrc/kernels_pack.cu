// PACK and UNPACK kernels: pure data movement, HBM-bound.
//
// pack: one warp per 32-particle chunk of a block (one side of one task).  The warp
//   (1) stages the pieces of the substruct arrays that hold the requested fields into shared memory with
//       coalesced cp.async (16 bytes when the stride allows, else 8 or 4; for power-of-two strides only the
//       16-byte pieces that are needed: for the 128-byte AoS record that is the difference between touching 2
//       and 4 sectors), particle 0 of the chunk always landing at the same staging offset;
//   (2) pre-pass, one lane per particle: x -> f32(x - frame) in place (one f64 subtraction, one RN conversion);
//   (3) re-slices the staging area into the compact record stream, 16 bytes per lane and store.  Which staging
//       word feeds which output word is the same for every chunk, so each lane computes its map once per launch.
//
// unpack: one warp per 32-particle chunk of a CELL.  The warp walks the cell's blocks in ascending (task, side)
// order, reading each block's slice with coalesced 16-byte loads (a round of independent loads in flight before
// the first add), and applies the per-field operator in f32 in that order (bit-reproducible, no atomics, no races:
// a particle is owned by exactly one warp per launch); the store fields are read and written once per launch.
#include <algorithm>

#include "internal.h"

namespace sph {

namespace {

constexpr int kPackWarps = 8;
constexpr int kUnpackWarps = 4;

template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem, const void* gmem) {
    if constexpr (BYTES == 16)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem));
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem), "n"(BYTES));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void st_stream16(void* p, uint4 v) {   // records are written once and read by another kernel
    asm volatile("st.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

template <int NIT>
__global__ void __launch_bounds__(kPackWarps * 32)
pack_kernel(Program prog, const CellChunk* __restrict__ cell_chunks, const uint32_t* __restrict__ occ_off128,
            const double* __restrict__ occ_frames, uint32_t n_cell_chunks, uint32_t slices, char* __restrict__ buf) {
    extern __shared__ __align__(16) unsigned char smem[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t R = prog.rec_words;
    const uint32_t templ_bytes = 128 * R;                           // 32 records
    unsigned char* stage = smem + (size_t)warp * (prog.smem_per_warp + 2 * templ_bytes);
    unsigned char* templ = stage + prog.smem_per_warp;              // two copies, used alternately

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

    const uint32_t n_items = n_cell_chunks * slices;
    for (uint32_t item = blockIdx.x * kPackWarps + warp; item < n_items; item += gridDim.x * kPackWarps) {
        const uint32_t cc = item / slices, sl = item - cc * slices;
        const CellChunk ch = cell_chunks[cc];
        const uint32_t per = (ch.nocc + slices - 1) / slices;
        const uint32_t ob = sl * per, oe = min(ch.nocc, ob + per);
        if (ob >= oe) continue;
        const uint32_t n = ch.count;
        // first occurrence's block offset and frame: in flight while the chunk is staged
        uint32_t o128 = __ldg(occ_off128 + ch.occ0 + ob);
        double f0 = 0., f1 = 0., f2 = 0.;
        if (prog.xrel) {
            const double* f = occ_frames + 3 * (size_t)(ch.occ0 + ob);
            f0 = __ldg(f); f1 = __ldg(f + 1); f2 = __ldg(f + 2);
        }

        // (1) stage the chunk's structs (once per item, not once per occurrence)
        for (uint32_t u = 0; u < prog.n_sub_used; ++u) {
            const PackSub su = prog.su[u];
            const char* g = su.base + (uint64_t)ch.first * su.stride;
            unsigned char* dst = stage + su.smem_base;
            const uint32_t nbytes = n * su.stride;
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
        cp_async_wait_all();
        __syncwarp();

        // (2) one lane per particle: keep x in registers (it is re-based for every occurrence); widen time_bin
        double x0 = 0., x1 = 0., x2 = 0.;
        if (prog.xrel && lane < n) {
            const unsigned char* px = stage + prog.x_src + lane * prog.x_stride;
            x0 = *reinterpret_cast<const double*>(px); x1 = *reinterpret_cast<const double*>(px + 8); x2 = *reinterpret_cast<const double*>(px + 16);
        }
        if (prog.tb && lane < n)
            *reinterpret_cast<uint32_t*>(stage + prog.tb_dst + 4 * lane) = stage[prog.tb_src + lane * prog.tb_stride];
        __syncwarp();

        // (3) re-slice the staging area into the record stream (both template copies); the x words are patched below
        const uint32_t nvec_out = (n * R + 3) >> 2;   // a last partial vector spills into the block's pad bytes
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const uint32_t v = lane + 32 * it;
            if (v < 8 * R) {
                uint4 o;
                o.x = *reinterpret_cast<const uint32_t*>(stage + src[it][0]);
                o.y = *reinterpret_cast<const uint32_t*>(stage + src[it][1]);
                o.z = *reinterpret_cast<const uint32_t*>(stage + src[it][2]);
                o.w = *reinterpret_cast<const uint32_t*>(stage + src[it][3]);
                *reinterpret_cast<uint4*>(templ + 16 * v) = o;
                *reinterpret_cast<uint4*>(templ + templ_bytes + 16 * v) = o;
            }
        }
        __syncwarp();   // the x words written here are overwritten by other lanes below

        // (4) one copy of the template per occurrence of the cell (task side), x re-based to that side's frame
        const uint64_t chunk_off = (uint64_t)ch.k0 * R * 4 + 16 * lane;
        for (uint32_t o = ob; o < oe; ++o) {
            unsigned char* T = templ + ((o - ob) & 1) * templ_bytes;
            char* out = buf + (uint64_t)o128 * 128 + chunk_off;
            if (prog.xrel && lane < n) {
                float* rec = reinterpret_cast<float*>(T) + lane * R;
                if (xw0 != 0xFFFFFFFFu) rec[xw0] = __double2float_rn(__dsub_rn(x0, f0));
                if (xw1 != 0xFFFFFFFFu) rec[xw1] = __double2float_rn(__dsub_rn(x1, f1));
                if (xw2 != 0xFFFFFFFFu) rec[xw2] = __double2float_rn(__dsub_rn(x2, f2));
            }
            if (o + 1 < oe) {   // next occurrence's table entries, in flight during this copy
                o128 = __ldg(occ_off128 + ch.occ0 + o + 1);
                if (prog.xrel) {
                    const double* f = occ_frames + 3 * (size_t)(ch.occ0 + o + 1);
                    f0 = __ldg(f); f1 = __ldg(f + 1); f2 = __ldg(f + 2);
                }
            }
            __syncwarp();
#pragma unroll
            for (int it = 0; it < NIT; ++it) {
                const uint32_t v = lane + 32 * it;
                if (v < nvec_out) st_stream16(out + 512 * it, *reinterpret_cast<const uint4*>(T + 16 * v));
            }
        }
        __syncwarp();   // staging and templates are reused by the next item
    }
}

// ---------------------------------------------------------------------------------------------------------

// One warp per 32-particle chunk of a cell.
//  (1) fetch: the chunk's slice of every block the cell occurs in (up to `slots` per round, normally all of them) is
//      copied into the warp's shared-memory ring with 16-byte cp.async -- no registers are held while the loads are
//      in flight, so a warp keeps 14-17 KB outstanding and an SM close to 200 KB;
//  (2) reduce: one lane per particle walks the slices in ascending (task, side) order.  With the lane owning a
//      record, the operator of word j (+=, max, =) is the same in every lane: no per-lane dispatch, no divergence.
//      Records are read with VEC-word shared loads (stride = record length: conflict-free when R / VEC is odd).
//  Words are processed in groups of GW; a record longer than GW keeps its running values in a scratch slot.
// The descriptor and block-offset table of the warp's next chunk are fetched while the current slices are in flight.
template <int VEC, int GW>
__global__ void __launch_bounds__(kUnpackWarps * 32)
unpack_kernel(StoreView view, Program prog, const CellChunk* __restrict__ cell_chunks, const uint32_t* __restrict__ occ_off128,
              uint32_t n_cell_chunks, const char* __restrict__ buf, uint32_t slots, uint32_t last_only, uint32_t all_sum) {
    extern __shared__ __align__(16) unsigned char smem[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t R = prog.rec_words;
    const uint32_t slot_bytes = 128 * R;
    const bool single = R <= GW;                       // the whole record lives in registers; else slot 0 is the scratch
    unsigned char* wbase = smem + (size_t)warp * (slots + (single ? 0u : 1u)) * slot_bytes;
    float* scratch = reinterpret_cast<float*>(wbase);  // [R][32]
    unsigned char* ring = wbase + (single ? 0u : slot_bytes);

    auto rounds_of = [&](const CellChunk& c, uint32_t* o_begin, uint32_t* per_round) {
        *o_begin = last_only ? c.nocc - 1 : 0;
        const uint32_t n_o = c.nocc - *o_begin, n_rounds = (n_o + slots - 1) / slots;
        *per_round = (n_o + n_rounds - 1) / n_rounds;                     // <= slots <= 32
    };
    auto first_table = [&](const CellChunk& c) {
        uint32_t o_begin, per_round;
        rounds_of(c, &o_begin, &per_round);
        return lane < min(per_round, c.nocc - o_begin) ? __ldg(occ_off128 + c.occ0 + o_begin + lane) : 0u;
    };
    // store access of word w of the lane's particle p
    auto word_addr = [&](uint32_t w, uint64_t p) { return view.base[prog.word[w].sub] + p * prog.word[w].stride + prog.word[w].a; };
    auto is_reduced = [&](uint32_t w) { return prog.word[w].kind == W_SUM || prog.word[w].kind == W_MAX; };

    // one group of words [g0, g0 + nw) reduced over the `lim` slices of the ring, in slice order
    auto reduce_group = [&](float (&acc)[GW], uint32_t g0, uint32_t nw, uint32_t lim) {
        const unsigned char* rec = ring + (lane * R + g0) * 4;
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

    const uint32_t cc_step = gridDim.x * kUnpackWarps;
    uint32_t cc = blockIdx.x * kUnpackWarps + warp;
    CellChunk ch_next{};
    uint32_t tbl_next = 0;
    if (cc < n_cell_chunks) { ch_next = cell_chunks[cc]; tbl_next = first_table(ch_next); }
    for (; cc < n_cell_chunks; cc += cc_step) {
        const CellChunk ch = ch_next;
        const uint32_t tbl_first = tbl_next;
        const uint32_t nvec = (ch.count * R + 3) >> 2;
        const char* slice = buf + (uint64_t)ch.k0 * R * 4 + 16 * lane;
        const bool live = lane < ch.count;
        const uint64_t p = (uint64_t)ch.first + lane;
        uint32_t o_begin, per_round;
        rounds_of(ch, &o_begin, &per_round);

        // running values: the store's own for the reduced words (issued before the slices are waited for)
        float acc[GW];
        if (single) {
#pragma unroll
            for (int j = 0; j < GW; ++j) acc[j] = 0.f;
#pragma unroll
            for (int j = 0; j < GW; ++j) {
                if ((uint32_t)j >= R || !live) continue;
                if (j % 4 == 0 && j + 3 < GW && prog.vec4[j]) {
                    const float4 t = *reinterpret_cast<const float4*>(word_addr(j, p));
                    acc[j] = t.x; if (j + 1 < GW) acc[j + 1] = t.y; if (j + 2 < GW) acc[j + 2] = t.z; if (j + 3 < GW) acc[j + 3] = t.w;
                } else if (!(j >= 4 * (j / 4) && prog.vec4[4 * (j / 4)] && 4 * (j / 4) + 3 < GW) && is_reduced(j)) {
                    acc[j] = *reinterpret_cast<const float*>(word_addr(j, p));
                }
            }
        } else {
            for (uint32_t w = 0; w < R; ++w)
                scratch[w * 32 + lane] = live && is_reduced(w) ? *reinterpret_cast<const float*>(word_addr(w, p)) : 0.f;
        }

        for (uint32_t ob = o_begin; ob < ch.nocc; ob += per_round) {
            const uint32_t lim = min(per_round, ch.nocc - ob);
            const uint32_t tbl = ob == o_begin ? tbl_first : (lane < lim ? __ldg(occ_off128 + ch.occ0 + ob + lane) : 0u);
            for (uint32_t u = 0; u < lim; ++u) {
                const char* src = slice + (uint64_t)__shfl_sync(0xFFFFFFFFu, tbl, u) * 128;
                unsigned char* dst = ring + u * slot_bytes + 16 * lane;
                for (uint32_t v = lane; v < nvec; v += 32, src += 512, dst += 512) cp_async<16>(dst, src);
            }
            if (ob == o_begin && cc + cc_step < n_cell_chunks) {   // next chunk's tables, while this chunk's slices are in flight
                ch_next = cell_chunks[cc + cc_step];
                tbl_next = first_table(ch_next);
            }
            cp_async_wait_all();
            __syncwarp();
            if (single) {
                reduce_group(acc, 0, R, lim);
            } else {
                for (uint32_t g0 = 0; g0 < R; g0 += GW) {
                    const uint32_t nw = min((uint32_t)GW, R - g0);
                    float a2[GW];
#pragma unroll
                    for (int j = 0; j < GW; ++j) a2[j] = (uint32_t)j < nw ? scratch[(g0 + j) * 32 + lane] : 0.f;
                    reduce_group(a2, g0, nw, lim);
#pragma unroll
                    for (int j = 0; j < GW; ++j) if ((uint32_t)j < nw) scratch[(g0 + j) * 32 + lane] = a2[j];
                }
            }
            __syncwarp();     // the ring is refilled by the next round / the next chunk
        }

        if (!live) continue;
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
}

// ---------------------------------------------------------------------------------------------------------

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

int g_sms = 0;
int32_t sm_count(int* out) {
    if (!g_sms) {
        int dev = 0;
        SPH_CUDA_TRY(cudaGetDevice(&dev));
        SPH_CUDA_TRY(cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, dev));
    }
    *out = g_sms;
    return SPH_OK;
}

template <int NIT>
int32_t launch_pack_nit(const sph_batch* b, const Program& prog, const uint32_t* d_occ_off128, char* d_buf, size_t smem, int sms, cudaStream_t st) {
    static size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        SPH_CUDA_TRY(cudaFuncSetAttribute(pack_kernel<NIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured = smem;
    }
    // resident CTAs per SM (shared memory and 64 warps bound it); a cell's occurrences are split into `slices` items
    // when there are fewer cell chunks than about two rounds of resident warps
    const uint32_t per_sm = (uint32_t)std::max<size_t>(1, std::min<size_t>(64 / kPackWarps, (220 * 1024) / (smem + 1024)));
    const uint32_t resident_warps = (uint32_t)sms * per_sm * kPackWarps;
    const uint32_t slices = std::min(8u, std::max(1u, (2 * resident_warps + b->n_cell_chunks - 1) / b->n_cell_chunks));
    const uint64_t items = (uint64_t)b->n_cell_chunks * slices;
    const uint32_t grid = (uint32_t)std::min<uint64_t>((items + kPackWarps - 1) / kPackWarps, (uint64_t)sms * per_sm);
    pack_kernel<NIT><<<grid, kPackWarps * 32, smem, st>>>(prog, b->d_cell_chunks, d_occ_off128, b->d_occ_frames, b->n_cell_chunks, slices, d_buf);
    return SPH_OK;
}

constexpr uint32_t kUnpackRingBytes = 17408;   // per warp: 27 slices of 32 x 20-byte records fit (a cell of a periodic grid occurs 27 times)

template <int VEC, int GW>
int32_t launch_unpack_t(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_occ_off128, const char* d_buf,
                        bool last_only, bool all_sum, int sms, cudaStream_t st) {
    const uint32_t slot_bytes = 128 * prog.rec_words;
    const uint32_t extra = prog.rec_words <= (uint32_t)GW ? 0 : 1;      // scratch slot of a long record
    const uint32_t slots = last_only ? 1u : std::max(1u, std::min(std::min(32u, b->max_nocc), kUnpackRingBytes / slot_bytes));
    const size_t smem = (size_t)kUnpackWarps * (slots + extra) * slot_bytes;
    static size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        SPH_CUDA_TRY(cudaFuncSetAttribute(unpack_kernel<VEC, GW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured = smem;
    }
    const uint32_t per_sm = (uint32_t)std::max<size_t>(1, std::min<size_t>(16, (227 * 1024) / (smem + 1024)));
    const uint32_t want = (b->n_cell_chunks + kUnpackWarps - 1) / kUnpackWarps;
    const uint32_t grid = std::min(want, (uint32_t)sms * per_sm);
    unpack_kernel<VEC, GW><<<grid, kUnpackWarps * 32, smem, st>>>(view, prog, b->d_cell_chunks, d_occ_off128, b->n_cell_chunks, d_buf, slots,
                                                                   last_only ? 1u : 0u, all_sum ? 1u : 0u);
    return SPH_OK;
}

}  // namespace

int32_t launch_pack(const StoreView& view, const sph_batch* b, const Program& prog_in, const uint32_t* d_occ_off128, char* d_buf, cudaStream_t st) {
    if (b->n_cell_chunks == 0) return SPH_OK;
    Program prog = prog_in;
    for (uint32_t u = 0; u < prog.n_sub_used; ++u) prog.su[u].base = view.base[prog.su[u].sub];
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    const size_t smem = ((size_t)prog.smem_per_warp + 2 * 128 * (size_t)prog.rec_words) * kPackWarps;
    if (smem > 200 * 1024) return fail(SPH_ERR_UNSUPPORTED, "layout needs %zu bytes of staging per CTA", smem);
    const uint32_t nit = (prog.rec_words + 3) / 4;   // 16-byte vectors per lane for a full chunk: ceil(32 R / 4 / 32)
    int32_t rc;
    if (nit <= 1) rc = launch_pack_nit<1>(b, prog, d_occ_off128, d_buf, smem, sms, st);
    else if (nit <= 2) rc = launch_pack_nit<2>(b, prog, d_occ_off128, d_buf, smem, sms, st);
    else if (nit <= 4) rc = launch_pack_nit<4>(b, prog, d_occ_off128, d_buf, smem, sms, st);
    else if (nit <= 6) rc = launch_pack_nit<6>(b, prog, d_occ_off128, d_buf, smem, sms, st);
    else if (nit <= 9) rc = launch_pack_nit<9>(b, prog, d_occ_off128, d_buf, smem, sms, st);
    else rc = launch_pack_nit<12>(b, prog, d_occ_off128, d_buf, smem, sms, st);
    if (rc) return rc;
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_unpack(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_occ_off128, const char* d_buf,
                      bool last_only, cudaStream_t st) {
    if (b->n_cell_chunks == 0) return SPH_OK;
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    bool all_sum = true;
    for (uint32_t w = 0; w < prog.rec_words; ++w) all_sum &= prog.word[w].kind == W_SUM;
    const uint32_t R = prog.rec_words;
    int32_t rc;
    if (R % 4 == 0) rc = R % 8 == 0 ? launch_unpack_t<4, 8>(view, b, prog, d_occ_off128, d_buf, last_only, all_sum, sms, st)
                                    : launch_unpack_t<4, 4>(view, b, prog, d_occ_off128, d_buf, last_only, all_sum, sms, st);
    else if (R % 2 == 0) rc = launch_unpack_t<2, 8>(view, b, prog, d_occ_off128, d_buf, last_only, all_sum, sms, st);
    else if (R % 5 == 0) rc = launch_unpack_t<1, 5>(view, b, prog, d_occ_off128, d_buf, last_only, all_sum, sms, st);
    else rc = launch_unpack_t<1, 8>(view, b, prog, d_occ_off128, d_buf, last_only, all_sum, sms, st);
    if (rc) return rc;
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
