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
__device__ __forceinline__ uint4 ld_once16(const void* p) {   // records are read exactly once: keep them out of L1
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}

template <int NIT>
__global__ void __launch_bounds__(kPackWarps * 32)
pack_kernel(Program prog, const SideRec* __restrict__ sides, const double* __restrict__ frames,
            const uint32_t* __restrict__ chunk_side, const uint32_t* __restrict__ off128, uint32_t n_chunks, char* __restrict__ buf) {
    extern __shared__ __align__(16) unsigned char smem[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned char* stage = smem + (size_t)warp * prog.smem_per_warp;
    const uint32_t R = prog.rec_words;

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

    for (uint32_t chunk = blockIdx.x * kPackWarps + warp; chunk < n_chunks; chunk += gridDim.x * kPackWarps) {
        const uint32_t side = chunk_side[chunk];
        const SideRec sr = sides[side];
        const uint32_t k0 = (chunk - sr.chunk0) * 32;
        const uint32_t n = min(32u, sr.count - k0);
        const uint64_t p0 = (uint64_t)sr.first + k0;
        const uint32_t o128 = off128[side];

        // (1) stage
        for (uint32_t u = 0; u < prog.n_sub_used; ++u) {
            const PackSub su = prog.su[u];
            const char* g = su.base + p0 * su.stride;
            unsigned char* dst = stage + su.smem_base;
            const uint32_t nbytes = n * su.stride;
            if (su.gran == 16) {
                const uint32_t nvec = nbytes >> 4;
                if (su.mask == 0xFFFFFFFFu) {
                    for (uint32_t v = lane; v < nvec; v += 32) cp_async<16>(dst + 16 * v, g + 16 * v);
                } else {
                    const uint32_t per = su.stride >> 4;
                    for (uint32_t v = lane; v < nvec; v += 32)
                        if (su.mask >> (v & (per - 1)) & 1) cp_async<16>(dst + 16 * v, g + 16 * v);
                }
            } else if (su.gran == 8) {
                for (uint32_t v = lane; v < (nbytes >> 3); v += 32) cp_async<8>(dst + 8 * v, g + 8 * v);
            } else {
                for (uint32_t v = lane; v < (nbytes >> 2); v += 32) cp_async<4>(dst + 4 * v, g + 4 * v);
            }
        }
        cp_async_wait_all();
        __syncwarp();

        // (2) pre-pass (each lane touches only its own particle's bytes)
        if (prog.xrel && lane < n) {
            unsigned char* px = stage + prog.x_src + lane * prog.x_stride;
            const double x0 = *reinterpret_cast<const double*>(px), x1 = *reinterpret_cast<const double*>(px + 8),
                         x2 = *reinterpret_cast<const double*>(px + 16);
            const double* f = frames + 3 * (size_t)side;
            const float r0 = __double2float_rn(__dsub_rn(x0, f[0])), r1 = __double2float_rn(__dsub_rn(x1, f[1])),
                        r2 = __double2float_rn(__dsub_rn(x2, f[2]));
            *reinterpret_cast<float2*>(px) = make_float2(r0, r1);
            *reinterpret_cast<float*>(px + 8) = r2;
        }
        if (prog.tb && lane < n)
            *reinterpret_cast<uint32_t*>(stage + prog.tb_dst + 4 * lane) = stage[prog.tb_src + lane * prog.tb_stride];
        __syncwarp();

        // (3) re-slice into records
        char* out = buf + (uint64_t)o128 * 128 + (uint64_t)k0 * R * 4;
        const uint32_t nvec_out = (n * R + 3) >> 2;   // a last partial vector spills into the block's pad bytes
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const uint32_t v = lane + 32 * it;
            if (v < nvec_out) {
                uint4 o;
                o.x = *reinterpret_cast<const uint32_t*>(stage + src[it][0]);
                o.y = *reinterpret_cast<const uint32_t*>(stage + src[it][1]);
                o.z = *reinterpret_cast<const uint32_t*>(stage + src[it][2]);
                o.w = *reinterpret_cast<const uint32_t*>(stage + src[it][3]);
                *reinterpret_cast<uint4*>(out + 16 * v) = o;
            }
        }
        __syncwarp();   // the staging region is reused by the next chunk
    }
}

// ---------------------------------------------------------------------------------------------------------

// meta word of the hoisted unpack map: store byte offset relative to the chunk's first particle | sub << 20 | kind << 24
__device__ __forceinline__ char* word_ptr(const StoreView* s_view, uint32_t meta, uint64_t first) {
    const uint32_t sub = (meta >> 20) & 0xF;
    return s_view->base[sub] + first * s_view->stride[sub] + (meta & 0xFFFFF);
}

template <int NIT, bool kLastOnly>
__global__ void __launch_bounds__(kUnpackWarps * 32)
unpack_kernel(StoreView view, Program prog, const CellChunk* __restrict__ cell_chunks, const uint32_t* __restrict__ occ_off128,
              uint32_t n_cell_chunks, const char* __restrict__ buf) {
    constexpr int UNR = NIT >= 8 ? 1 : (NIT >= 4 ? 2 : (NIT >= 2 ? 4 : 8));   // blocks whose records are in flight together
    __shared__ StoreView s_view;     // indexed per lane (the substruct differs from word to word)
    if (threadIdx.x == 0) s_view = view;
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t R = prog.rec_words;
    uint32_t meta[NIT][4];
#pragma unroll
    for (int it = 0; it < NIT; ++it)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t g = 4 * (lane + 32 * it) + j;
            const uint32_t k = g / R, w = g - k * R;
            meta[it][j] = k < 32 ? (k * prog.word[w].stride + prog.word[w].a) | (uint32_t)prog.word[w].sub << 20 | (uint32_t)prog.word[w].kind << 24
                                 : (uint32_t)W_SKIP << 24;
        }

    for (uint32_t cc = blockIdx.x * kUnpackWarps + warp; cc < n_cell_chunks; cc += gridDim.x * kUnpackWarps) {
        const CellChunk ch = cell_chunks[cc];
        const uint32_t total = ch.count * R, nvec = (total + 3) >> 2;
        const char* slice = buf + (uint64_t)ch.k0 * R * 4 + 16 * lane;
        float acc[NIT][4];
        uint32_t kind[NIT][4];
#pragma unroll
        for (int it = 0; it < NIT; ++it)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t g = 4 * (lane + 32 * it) + j;
                kind[it][j] = g < total ? meta[it][j] >> 24 : (uint32_t)W_SKIP;
                acc[it][j] = 0.f;
                if (!kLastOnly && (kind[it][j] == W_SUM || kind[it][j] == W_MAX))
                    acc[it][j] = *reinterpret_cast<const float*>(word_ptr(&s_view, meta[it][j], ch.first));
            }
        for (uint32_t ob = kLastOnly ? ch.nocc - 1 : 0; ob < ch.nocc; ob += 32) {
            const uint32_t lim = min(32u, ch.nocc - ob);
            const uint32_t tbl = lane < lim ? occ_off128[ch.occ0 + ob + lane] : 0;
            for (uint32_t u0 = 0; u0 < lim; u0 += UNR) {
                uint4 r[UNR][NIT];
#pragma unroll
                for (int u = 0; u < UNR; ++u) {
                    const uint32_t o128 = __shfl_sync(0xFFFFFFFFu, tbl, (u0 + u) & 31);
                    if (u0 + u < lim) {
#pragma unroll
                        for (int it = 0; it < NIT; ++it)
                            if (lane + 32 * it < nvec) r[u][it] = ld_once16(slice + (uint64_t)o128 * 128 + 512 * it);
                    }
                }
#pragma unroll
                for (int u = 0; u < UNR; ++u) {
                    if (u0 + u < lim) {
#pragma unroll
                        for (int it = 0; it < NIT; ++it) {
                            const float rv[4] = {__uint_as_float(r[u][it].x), __uint_as_float(r[u][it].y), __uint_as_float(r[u][it].z),
                                                 __uint_as_float(r[u][it].w)};
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                const float s = __fadd_rn(acc[it][j], rv[j]), m = fmaxf(acc[it][j], rv[j]);
                                acc[it][j] = kind[it][j] == W_SUM ? s : (kind[it][j] == W_MAX ? m : rv[j]);
                            }
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int it = 0; it < NIT; ++it)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (kind[it][j] == W_SKIP) continue;
                char* dst = word_ptr(&s_view, meta[it][j], ch.first);
                if (kind[it][j] == W_ASSIGN_BYTE) *reinterpret_cast<unsigned char*>(dst) = (unsigned char)__float_as_uint(acc[it][j]);
                else *reinterpret_cast<float*>(dst) = acc[it][j];
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
int32_t launch_pack_nit(const sph_batch* b, const Program& prog, const uint32_t* d_off128, char* d_buf,
                        uint32_t grid, size_t smem, cudaStream_t st) {
    static size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        SPH_CUDA_TRY(cudaFuncSetAttribute(pack_kernel<NIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured = smem;
    }
    pack_kernel<NIT><<<grid, kPackWarps * 32, smem, st>>>(prog, b->d_sides, b->d_frames, b->d_chunk_side, d_off128, b->n_chunks, d_buf);
    return SPH_OK;
}

template <int NIT>
void launch_unpack_nit(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_occ_off128, const char* d_buf,
                       bool last_only, uint32_t grid, cudaStream_t st) {
    if (last_only)
        unpack_kernel<NIT, true><<<grid, kUnpackWarps * 32, 0, st>>>(view, prog, b->d_cell_chunks, d_occ_off128, b->n_cell_chunks, d_buf);
    else
        unpack_kernel<NIT, false><<<grid, kUnpackWarps * 32, 0, st>>>(view, prog, b->d_cell_chunks, d_occ_off128, b->n_cell_chunks, d_buf);
}

}  // namespace

int32_t launch_pack(const StoreView& view, const sph_batch* b, const Program& prog_in, const uint32_t* d_off128, char* d_buf, cudaStream_t st) {
    if (b->n_chunks == 0) return SPH_OK;
    Program prog = prog_in;
    for (uint32_t u = 0; u < prog.n_sub_used; ++u) prog.su[u].base = view.base[prog.su[u].sub];
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    const size_t smem = (size_t)prog.smem_per_warp * kPackWarps;
    if (smem > 200 * 1024) return fail(SPH_ERR_UNSUPPORTED, "layout needs %zu bytes of staging per CTA", smem);
    const uint32_t want = (b->n_chunks + kPackWarps - 1) / kPackWarps;
    const uint32_t grid = min(want, (uint32_t)sms * 8);
    const uint32_t nit = (prog.rec_words + 3) / 4;   // 16-byte vectors per lane for a full chunk: ceil(32 R / 4 / 32)
    int32_t rc;
    if (nit <= 1) rc = launch_pack_nit<1>(b, prog, d_off128, d_buf, grid, smem, st);
    else if (nit <= 2) rc = launch_pack_nit<2>(b, prog, d_off128, d_buf, grid, smem, st);
    else if (nit <= 4) rc = launch_pack_nit<4>(b, prog, d_off128, d_buf, grid, smem, st);
    else if (nit <= 6) rc = launch_pack_nit<6>(b, prog, d_off128, d_buf, grid, smem, st);
    else if (nit <= 9) rc = launch_pack_nit<9>(b, prog, d_off128, d_buf, grid, smem, st);
    else rc = launch_pack_nit<12>(b, prog, d_off128, d_buf, grid, smem, st);
    if (rc) return rc;
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_unpack(const StoreView& view, const sph_batch* b, const Program& prog, const uint32_t* d_occ_off128, const char* d_buf,
                      bool last_only, cudaStream_t st) {
    if (b->n_cell_chunks == 0) return SPH_OK;
    int sms = 0;
    if (int32_t rc = sm_count(&sms)) return rc;
    const uint32_t want = (b->n_cell_chunks + kUnpackWarps - 1) / kUnpackWarps;
    const uint32_t grid = min(want, (uint32_t)sms * 16);
    const uint32_t nit = (prog.rec_words + 3) / 4;
    if (nit <= 1) launch_unpack_nit<1>(view, b, prog, d_occ_off128, d_buf, last_only, grid, st);
    else if (nit <= 2) launch_unpack_nit<2>(view, b, prog, d_occ_off128, d_buf, last_only, grid, st);
    else if (nit <= 4) launch_unpack_nit<4>(view, b, prog, d_occ_off128, d_buf, last_only, grid, st);
    else if (nit <= 6) launch_unpack_nit<6>(view, b, prog, d_occ_off128, d_buf, last_only, grid, st);
    else if (nit <= 9) launch_unpack_nit<9>(view, b, prog, d_occ_off128, d_buf, last_only, grid, st);
    else launch_unpack_nit<12>(view, b, prog, d_occ_off128, d_buf, last_only, grid, st);
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
