// PACK and UNPACK kernels: pure data movement, HBM-bound.
//
// pack: one warp per 32-particle chunk of a block.  The warp (1) stages the 16-byte pieces of the substruct
// arrays that hold the requested fields into shared memory with coalesced cp.async (only the pieces that are
// needed: for the 128-byte AoS record that is the difference between touching 2 and 4 sectors), then
// (2) re-slices them into the compact record stream and writes it with coalesced 16-byte stores.
//
// unpack: one warp per 32-particle chunk of a CELL.  The warp walks the cell's blocks in ascending task order,
// reading each block's slice with coalesced 16-byte loads, and applies the per-field operator in f32 in that
// order (bit-reproducible, no atomics, no races: a particle is owned by exactly one warp per launch); the store
// fields are read and written once per launch.
#include "internal.h"

namespace sph {

namespace {

constexpr int kPackWarps = 8;
constexpr int kUnpackWarps = 8;

struct SWord {          // word descriptor as the kernels use it (shared memory copy)
    uint32_t a;         // pack: staging byte offset of the word inside the warp's region (without the per-chunk shift)
                        // unpack: byte offset inside the substruct
    uint32_t b;         // stride | kind << 16 | dim << 20 | used_idx << 24
};

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void st_stream16(void* p, const uint4& v) {
    asm volatile("st.global.cs.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ uint4 ld_stream16(const void* p) {
    uint4 v;
    asm volatile("ld.global.cs.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}

__global__ void __launch_bounds__(kPackWarps * 32)
pack_kernel(StoreView view, Program prog, const SideRec* __restrict__ sides, const double* __restrict__ frames,
            const uint32_t* __restrict__ chunk_side, const uint32_t* __restrict__ off128, uint32_t n_chunks, char* __restrict__ buf) {
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ SWord s_word[kMaxRecWords];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (uint32_t w = threadIdx.x; w < prog.rec_words; w += blockDim.x) {
        const WordDesc wd = prog.word[w];
        s_word[w].a = prog.smem_base[wd.used_idx] + wd.off;
        s_word[w].b = view.stride[wd.sub] | (uint32_t)wd.kind << 16 | (uint32_t)wd.dim << 20 | (uint32_t)wd.used_idx << 24;
    }
    __syncthreads();
    unsigned char* stage = smem + (size_t)warp * prog.smem_per_warp;
    const uint32_t rec_words = prog.rec_words;

    for (uint32_t chunk = blockIdx.x * kPackWarps + warp; chunk < n_chunks; chunk += gridDim.x * kPackWarps) {
        const uint32_t side = chunk_side[chunk];
        const SideRec sr = sides[side];
        const uint32_t k0 = (chunk - sr.chunk0) * 32;
        const uint32_t n = min(32u, sr.count - k0);
        const uint64_t p0 = (uint64_t)sr.first + k0;

        // (1) stage the needed 16-byte pieces of every substruct the record draws from
        for (uint32_t u = 0; u < prog.n_sub_used; ++u) {
            const uint32_t s = prog.sub_used[u], stride = view.stride[s], mask = prog.chunk_mask[u];
            const uint64_t byte0 = p0 * stride;
            const uint64_t a0 = byte0 & ~15ull;
            const uint32_t nvec = (uint32_t)(((byte0 + (uint64_t)n * stride + 15) & ~15ull) - a0) >> 4;
            const char* src = view.base[s] + a0;
            unsigned char* dst = stage + prog.smem_base[u];
            if (mask == 0xFFFFFFFFu) {
                for (uint32_t v = lane; v < nvec; v += 32) cp_async16(dst + 16 * v, src + 16 * v);
            } else {   // power-of-two stride: skip the pieces no requested field lives in
                const uint32_t per = stride >> 4;
                for (uint32_t v = lane; v < nvec; v += 32)
                    if (mask >> (v & (per - 1)) & 1) cp_async16(dst + 16 * v, src + 16 * v);
            }
        }
        cp_async_wait_all();
        __syncwarp();

        // (2) re-slice into records
        const double fx = frames[3 * side], fy = frames[3 * side + 1], fz = frames[3 * side + 2];
        char* out = buf + (uint64_t)off128[side] * 128 + (uint64_t)k0 * rec_words * 4;
        const uint32_t total = n * rec_words, nvec_out = (total + 3) >> 2;
        for (uint32_t v = lane; v < nvec_out; v += 32) {
            uint32_t o[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t g = 4 * v + j;
                const uint32_t k = (g * prog.div_magic) >> 16;
                const uint32_t w = g - k * rec_words;
                const SWord sw = s_word[w];
                const uint32_t stride = sw.b & 0xFFFF, kind = (sw.b >> 16) & 0xF;
                const uint32_t shift = (uint32_t)(p0 * stride) & 15u;   // where particle 0 of the chunk sits in its staged piece
                const unsigned char* src = stage + sw.a + shift + k * stride;
                uint32_t val = 0;
                if (g < total) {
                    if (kind == W_COPY) {
                        val = *reinterpret_cast<const uint32_t*>(src);
                    } else if (kind == W_XREL) {
                        const uint2 raw = *reinterpret_cast<const uint2*>(src);
                        const uint32_t dim = (sw.b >> 20) & 0xF;
                        const double f = dim == 0 ? fx : (dim == 1 ? fy : fz);
                        val = __float_as_uint(__double2float_rn(__dsub_rn(__hiloint2double((int)raw.y, (int)raw.x), f)));
                    } else {   // W_TIMEBIN
                        val = *src;
                    }
                }
                o[j] = val;
            }
            st_stream16(out + 16 * v, make_uint4(o[0], o[1], o[2], o[3]));
        }
        __syncwarp();   // the staging region is reused by the next chunk
    }
}

// ---------------------------------------------------------------------------------------------------------

template <bool kLastOnly>
__global__ void __launch_bounds__(kUnpackWarps * 32)
unpack_kernel(StoreView view, Program prog, const SideRec* __restrict__ sides, const CellChunk* __restrict__ cell_chunks,
              const uint32_t* __restrict__ occ_side, const uint32_t* __restrict__ off128, uint32_t n_cell_chunks, const char* __restrict__ buf) {
    __shared__ SWord s_word[kMaxRecWords];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (uint32_t w = threadIdx.x; w < prog.rec_words; w += blockDim.x) {
        const WordDesc wd = prog.word[w];
        s_word[w].a = wd.off;
        s_word[w].b = view.stride[wd.sub] | (uint32_t)wd.kind << 16 | (uint32_t)wd.sub << 24;
    }
    __syncthreads();
    const uint32_t rec_words = prog.rec_words;

    for (uint32_t cc = blockIdx.x * kUnpackWarps + warp; cc < n_cell_chunks; cc += gridDim.x * kUnpackWarps) {
        const CellChunk ch = cell_chunks[cc];
        const uint32_t total = ch.count * rec_words, nvec = (total + 3) >> 2;
        const uint64_t slice = (uint64_t)ch.k0 * rec_words * 4;
        for (uint32_t v = lane; v < nvec; v += 32) {
            // the four record words this lane owns -> (particle, field word), store address, operator
            char* dst[4];
            uint32_t kind[4];
            float acc[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t g = 4 * v + j;
                const uint32_t k = (g * prog.div_magic) >> 16;
                const uint32_t w = g - k * rec_words;
                const SWord sw = s_word[w];
                const uint32_t stride = sw.b & 0xFFFF, sub = sw.b >> 24;
                kind[j] = g < total ? (sw.b >> 16) & 0xF : (uint32_t)W_SKIP;
                dst[j] = view.base[sub] + ((uint64_t)ch.first + k) * stride + sw.a;
                acc[j] = 0.f;
                if (kind[j] == W_SUM || kind[j] == W_MAX) acc[j] = *reinterpret_cast<const float*>(dst[j]);
            }
            uint32_t o = kLastOnly ? ch.nocc - 1 : 0;
#pragma unroll 4
            for (; o < ch.nocc; ++o) {
                const uint32_t side = occ_side[ch.occ0 + o];
                const uint4 r = ld_stream16(buf + (uint64_t)off128[side] * 128 + slice + 16 * v);
                const float rv[4] = {__uint_as_float(r.x), __uint_as_float(r.y), __uint_as_float(r.z), __uint_as_float(r.w)};
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    if (kind[j] == W_SUM) acc[j] = __fadd_rn(acc[j], rv[j]);
                    else if (kind[j] == W_MAX) acc[j] = fmaxf(acc[j], rv[j]);
                    else acc[j] = rv[j];
                }
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (kind[j] == W_SKIP) continue;
                if (kind[j] == W_ASSIGN_BYTE) *reinterpret_cast<unsigned char*>(dst[j]) = (unsigned char)__float_as_uint(acc[j]);
                else *reinterpret_cast<float*>(dst[j]) = acc[j];
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
        *reinterpret_cast<float*>(view.base[wd.sub] + p * view.stride[wd.sub] + wd.off) = 0.f;
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

}  // namespace

int32_t launch_pack(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_off128, char* d_buf, cudaStream_t st) {
    if (b->n_chunks == 0) return SPH_OK;
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    const size_t smem = (size_t)prog.smem_per_warp * kPackWarps;
    if (smem > 200 * 1024) return fail(SPH_ERR_UNSUPPORTED, "layout needs %zu bytes of staging per CTA", smem);
    static size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        SPH_CUDA_TRY(cudaFuncSetAttribute(pack_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured = smem;
    }
    const uint32_t want = (b->n_chunks + kPackWarps - 1) / kPackWarps;
    const uint32_t grid = min(want, (uint32_t)sms * 8);
    pack_kernel<<<grid, kPackWarps * 32, smem, st>>>(view, prog, b->d_sides, b->d_frames, b->d_chunk_side, d_off128, b->n_chunks, d_buf);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_unpack(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_off128, const char* d_buf,
                      bool last_only, cudaStream_t st) {
    if (b->n_cell_chunks == 0) return SPH_OK;
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    const uint32_t want = (b->n_cell_chunks + kUnpackWarps - 1) / kUnpackWarps;
    const uint32_t grid = min(want, (uint32_t)sms * 8);
    if (last_only)
        unpack_kernel<true><<<grid, kUnpackWarps * 32, 0, st>>>(view, prog, b->d_sides, b->d_cell_chunks, b->d_occ_side, d_off128, b->n_cell_chunks, d_buf);
    else
        unpack_kernel<false><<<grid, kUnpackWarps * 32, 0, st>>>(view, prog, b->d_sides, b->d_cell_chunks, b->d_occ_side, d_off128, b->n_cell_chunks, d_buf);
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
