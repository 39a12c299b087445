// DENSITY and FORCE interaction loops over cell / cell-pair tasks.
//
// Nothing here is a dense contraction (a few percent of the candidate pairs are neighbours and the per-pair
// work is a distance test), so this is plain FP32 ALU work, not tensor-core work.
//
// Work item = (32 target particles of one block) x (the block they gather from: the task's other side, or the
// block itself for a self task).  One warp per item, warps never wait for one another (no __syncthreads):
//   (a) the 32 target records are staged through shared memory with coalesced 16-byte loads; the warp reduces
//       their bounding box and largest h with shuffles;
//   (b) the source block is streamed 32 records at a time the same way; a source outside the targets' reach box
//       (box grown by 2 h_max, for the force loop by max(2 h_max, 2 h_j)) cannot be anybody's neighbour and is
//       dropped; the others are compacted (ballot + popc) into a 64-entry tile of float4s;
//   (c) phase 1, branch-free: every lane tests its target against every tile entry (broadcast LDS.128,
//       3 FADD + FMUL + 2 FFMA + compare) and records the outcome in a 64-bit hit mask;
//   (d) phase 2: every lane walks the set bits of its mask and evaluates the kernel terms for real neighbours only.
// Sums are accumulated per lane in tile order = source order, so results are bit-reproducible run to run.
#include "internal.h"

namespace sph {

namespace {

constexpr int kLoopWarps = 4;
constexpr int kTile = 64;                  // compacted sources per flush = bits in the per-lane hit mask
constexpr float kInvPi = 0.318309886183790671538f;
constexpr float kFar = 1.0e18f;            // coordinate of a tile pad entry / an idle lane: never within reach
constexpr float kReachSlack = 1.0f + 1.0e-4f;   // the reach box is a superset test; keep it clear of f32 rounding

__device__ __forceinline__ float warp_min(float v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fminf(v, __shfl_xor_sync(0xFFFFFFFFu, v, o));
    return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xFFFFFFFFu, v, o));
    return v;
}
__device__ __forceinline__ float sqrt_approx(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ uint32_t lanemask_lt() {
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// n records of `words` 4-byte words, contiguous and 16-byte aligned in global memory -> raw (shared), coalesced
__device__ __forceinline__ void stage_records(float* raw, const char* g, uint32_t n, uint32_t words, uint32_t lane) {
    const uint32_t nvec = (n * words + 3) >> 2;   // a last partial vector reads into the block's pad bytes
    for (uint32_t v = lane; v < nvec; v += 32) reinterpret_cast<uint4*>(raw)[v] = __ldg(reinterpret_cast<const uint4*>(g) + v);
}

// cubic spline (M4), q = r/h in [0, 2): value and derivative
__device__ __forceinline__ void spline(float q, float* w, float* dw) {
    const float t2 = 2.0f - q;
    const float w_in = fmaf(q * q, fmaf(0.75f, q, -1.5f), 1.0f);      // 1 - 1.5 q^2 + 0.75 q^3
    const float dw_in = q * fmaf(2.25f, q, -3.0f);                    // -3 q + 2.25 q^2
    const float w_out = 0.25f * t2 * t2 * t2, dw_out = -0.75f * t2 * t2;
    *w = q < 1.0f ? w_in : w_out;
    *dw = q < 1.0f ? dw_in : dw_out;
}
__device__ __forceinline__ float spline_dw(float q) {
    const float t2 = fmaxf(2.0f - q, 0.0f);
    return q < 1.0f ? q * fmaf(2.25f, q, -3.0f) : -0.75f * t2 * t2;
}

struct Item {
    uint32_t n_t, n_s, k0;
    const char *tin, *sin;
    char* tout;
};

template <int REC_IN, int REC_OUT>
__device__ __forceinline__ Item load_item(uint32_t item, const SideRec* __restrict__ sides, const uint32_t* __restrict__ chunk_side,
                                          const uint32_t* __restrict__ chunk_src, const uint32_t* __restrict__ off_in,
                                          const uint32_t* __restrict__ off_out, const char* in, char* out) {
    const uint32_t tgt = chunk_side[item], src = chunk_src[item];
    const SideRec st = sides[tgt];
    Item it;
    it.k0 = (item - st.chunk0) * 32;
    it.n_t = min(32u, st.count - it.k0);
    it.n_s = sides[src].count;
    it.tin = in + (uint64_t)off_in[tgt] * 128 + (uint64_t)it.k0 * REC_IN;
    it.sin = in + (uint64_t)off_in[src] * 128;
    it.tout = out + (uint64_t)off_out[tgt] * 128 + (uint64_t)it.k0 * REC_OUT;
    return it;
}

// ------------------------------------------------------------------------------------------------- density

struct DensityWarpSmem {
    float4 tile[kTile];      // x, y, z, m of the compacted sources
    float raw[32 * 5];       // staging of 32 DENSITY_IN records: xr0 xr1 xr2 h m
};

__global__ void __launch_bounds__(kLoopWarps * 32)
density_kernel(const SideRec* __restrict__ sides, const uint32_t* __restrict__ chunk_side, const uint32_t* __restrict__ chunk_src,
               const uint32_t* __restrict__ off_in, const uint32_t* __restrict__ off_out, const char* __restrict__ in,
               char* __restrict__ out, uint32_t n_items) {
    __shared__ __align__(16) DensityWarpSmem s_all[kLoopWarps];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    DensityWarpSmem& sm = s_all[warp];
    const uint32_t lt = lanemask_lt();

    for (uint32_t item = blockIdx.x * kLoopWarps + warp; item < n_items; item += gridDim.x * kLoopWarps) {
        const Item it = load_item<20, 16>(item, sides, chunk_side, chunk_src, off_in, off_out, in, out);
        stage_records(sm.raw, it.tin, it.n_t, 5, lane);
        __syncwarp();
        const bool valid = lane < it.n_t;
        const float xi = valid ? sm.raw[5 * lane] : -kFar, yi = valid ? sm.raw[5 * lane + 1] : -kFar, zi = valid ? sm.raw[5 * lane + 2] : -kFar;
        const float hi = valid ? sm.raw[5 * lane + 3] : 0.f;
        __syncwarp();
        const float hc2 = 4.0f * hi * hi, inv_h = valid ? 1.0f / hi : 0.f;
        const float reach = 2.0f * warp_max(hi) * kReachSlack;
        const float lox = warp_min(valid ? xi : kFar) - reach, hix = warp_max(xi) + reach;
        const float loy = warp_min(valid ? yi : kFar) - reach, hiy = warp_max(yi) + reach;
        const float loz = warp_min(valid ? zi : kFar) - reach, hiz = warp_max(zi) + reach;
        float s_mw = 0.f, s_mg = 0.f, s_w = 0.f, s_g = 0.f;     // sums of m w, m (3w + q w'), w, (3w + q w')

        auto flush = [&](uint32_t cnt) {
            const uint32_t n8 = (cnt + 7) & ~7u;
            if (lane < n8 - cnt) sm.tile[cnt + lane] = make_float4(kFar, kFar, kFar, 0.f);
            __syncwarp();
            uint32_t mlo = 0, mhi = 0;
            for (uint32_t j = 0; j < n8; j += 8) {
                uint32_t m8 = 0;
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const float4 s = sm.tile[j + u];
                    const float dx = xi - s.x, dy = yi - s.y, dz = zi - s.z;
                    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    m8 |= r2 < hc2 ? 1u << u : 0u;
                }
                if (j < 32) mlo |= m8 << j; else mhi |= m8 << (j - 32);
            }
            auto hit = [&](uint32_t j) {
                const float4 s = sm.tile[j];
                const float dx = xi - s.x, dy = yi - s.y, dz = zi - s.z;
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                const float q = sqrt_approx(r2) * inv_h;
                float w, dw;
                spline(q, &w, &dw);
                const float g = fmaf(q, dw, 3.0f * w);
                s_mw = fmaf(s.w, w, s_mw); s_mg = fmaf(s.w, g, s_mg);
                s_w += w; s_g += g;
            };
            while (mlo) { const uint32_t j = __ffs(mlo) - 1; mlo &= mlo - 1; hit(j); }
            while (mhi) { const uint32_t j = __ffs(mhi) - 1; mhi &= mhi - 1; hit(32 + j); }
            __syncwarp();
        };

        uint32_t cnt = 0;
        for (uint32_t j0 = 0; j0 < it.n_s; j0 += 32) {
            const uint32_t nj = min(32u, it.n_s - j0);
            stage_records(sm.raw, it.sin + (uint64_t)j0 * 20, nj, 5, lane);
            __syncwarp();
            float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
            bool ok = false;
            if (lane < nj) {
                s = make_float4(sm.raw[5 * lane], sm.raw[5 * lane + 1], sm.raw[5 * lane + 2], sm.raw[5 * lane + 4]);
                ok = s.x > lox && s.x < hix && s.y > loy && s.y < hiy && s.z > loz && s.z < hiz;
            }
            __syncwarp();
            const uint32_t ball = __ballot_sync(0xFFFFFFFFu, ok), c = __popc(ball);
            if (cnt + c > kTile) { flush(cnt); cnt = 0; }
            if (ok) sm.tile[cnt + __popc(ball & lt)] = s;
            cnt += c;
        }
        if (cnt) flush(cnt);
        if (valid) {
            const float n3 = kInvPi * inv_h * inv_h * inv_h, n4 = n3 * inv_h;
            reinterpret_cast<float4*>(it.tout)[lane] = make_float4(s_mw * n3, -s_mg * n4, s_w * n3, -s_g * n4);
        }
    }
}

// ------------------------------------------------------------------------------------------------- force

struct ForceWarpSmem {
    float4 ta[kTile];        // x, y, z, 4 h^2
    float4 tb[kTile];        // vx, vy, vz, m
    float4 tc[kTile];        // rho, A = P / (Omega rho^2), c_s, 1/h
    float raw[32 * 13];      // staging of 32 FORCE_IN records: xr0 xr1 xr2 h m rho rho_dh v0 v1 v2 u P cs (and of the 32 results)
};

__global__ void __launch_bounds__(kLoopWarps * 32)
force_kernel(const SideRec* __restrict__ sides, const uint32_t* __restrict__ chunk_side, const uint32_t* __restrict__ chunk_src,
             const uint32_t* __restrict__ off_in, const uint32_t* __restrict__ off_out, const char* __restrict__ in,
             char* __restrict__ out, uint32_t n_items, float alpha, float beta) {
    __shared__ __align__(16) ForceWarpSmem s_all[kLoopWarps];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ForceWarpSmem& sm = s_all[warp];
    const uint32_t lt = lanemask_lt();

    for (uint32_t item = blockIdx.x * kLoopWarps + warp; item < n_items; item += gridDim.x * kLoopWarps) {
        const Item it = load_item<52, 20>(item, sides, chunk_side, chunk_src, off_in, off_out, in, out);
        stage_records(sm.raw, it.tin, it.n_t, 13, lane);
        __syncwarp();
        const bool valid = lane < it.n_t;
        float xi = -kFar, yi = -kFar, zi = -kFar, hi = 0.f, rhoi = 1.f, rho_dhi = 0.f, vxi = 0.f, vyi = 0.f, vzi = 0.f, Pi = 0.f, ci = 0.f;
        if (valid) {
            const float* r = sm.raw + 13 * lane;
            xi = r[0]; yi = r[1]; zi = r[2]; hi = r[3]; rhoi = r[5]; rho_dhi = r[6]; vxi = r[7]; vyi = r[8]; vzi = r[9]; Pi = r[11]; ci = r[12];
        }
        __syncwarp();
        const float hc2i = 4.0f * hi * hi, inv_hi = valid ? 1.0f / hi : 0.f;
        const float n4i = kInvPi * (inv_hi * inv_hi) * (inv_hi * inv_hi);
        const float Ai = Pi / ((1.0f + hi * rho_dhi / (3.0f * rhoi)) * rhoi * rhoi);
        const float reach_t = 2.0f * warp_max(hi);
        const float lox = warp_min(valid ? xi : kFar), hix = warp_max(xi);
        const float loy = warp_min(valid ? yi : kFar), hiy = warp_max(yi);
        const float loz = warp_min(valid ? zi : kFar), hiz = warp_max(zi);
        float ax = 0.f, ay = 0.f, az = 0.f, du = 0.f, vsig = 0.f;

        auto flush = [&](uint32_t cnt) {
            const uint32_t n8 = (cnt + 7) & ~7u;
            if (lane < n8 - cnt) sm.ta[cnt + lane] = make_float4(kFar, kFar, kFar, 0.f);
            __syncwarp();
            uint32_t mlo = 0, mhi = 0;
            for (uint32_t j = 0; j < n8; j += 8) {
                uint32_t m8 = 0;
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const float4 a = sm.ta[j + u];
                    const float dx = xi - a.x, dy = yi - a.y, dz = zi - a.z;
                    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    m8 |= (r2 < fmaxf(hc2i, a.w) && r2 > 0.f) ? 1u << u : 0u;
                }
                if (j < 32) mlo |= m8 << j; else mhi |= m8 << (j - 32);
            }
            auto hit = [&](uint32_t j) {
                const float4 a = sm.ta[j], b = sm.tb[j], c = sm.tc[j];
                const float dx = xi - a.x, dy = yi - a.y, dz = zi - a.z;
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                float rinv = rsqrtf(r2);
                rinv = rinv * fmaf(-0.5f * r2 * rinv, rinv, 1.5f);      // one Newton step: ~1 ulp
                const float r = r2 * rinv;
                const float Gi = spline_dw(r * inv_hi) * n4i;
                const float ih2 = c.w * c.w;
                const float Gj = spline_dw(r * c.w) * (kInvPi * ih2 * ih2);
                const float vr = fmaf(vzi - b.z, dz, fmaf(vyi - b.y, dy, (vxi - b.x) * dx)) * rinv;
                const float mu = fminf(vr, 0.f);
                const float vs = fmaf(-beta, mu, ci + c.z);
                const float visc = -alpha * vs * mu * __frcp_rn(rhoi + c.x);   // -(alpha/2) vs mu / ((rho_i+rho_j)/2)
                const float vG = visc * 0.5f * (Gi + Gj);
                const float AG = Ai * Gi, BG = c.y * Gj;
                const float fr = -b.w * (AG + BG + vG) * rinv;
                ax = fmaf(fr, dx, ax); ay = fmaf(fr, dy, ay); az = fmaf(fr, dz, az);
                du = fmaf(b.w * fmaf(0.5f, vG, AG), vr, du);
                vsig = fmaxf(vsig, vs);
            };
            while (mlo) { const uint32_t j = __ffs(mlo) - 1; mlo &= mlo - 1; hit(j); }
            while (mhi) { const uint32_t j = __ffs(mhi) - 1; mhi &= mhi - 1; hit(32 + j); }
            __syncwarp();
        };

        uint32_t cnt = 0;
        for (uint32_t j0 = 0; j0 < it.n_s; j0 += 32) {
            const uint32_t nj = min(32u, it.n_s - j0);
            stage_records(sm.raw, it.sin + (uint64_t)j0 * 52, nj, 13, lane);
            __syncwarp();
            float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a, c = a;
            bool ok = false;
            if (lane < nj) {
                const float* r = sm.raw + 13 * lane;
                const float h = r[3], rho = r[5];
                const float reach = fmaxf(reach_t, 2.0f * h) * kReachSlack;
                a = make_float4(r[0], r[1], r[2], 4.0f * h * h);
                ok = a.x > lox - reach && a.x < hix + reach && a.y > loy - reach && a.y < hiy + reach && a.z > loz - reach && a.z < hiz + reach;
                if (ok) {
                    b = make_float4(r[7], r[8], r[9], r[4]);
                    c = make_float4(rho, r[11] / ((1.0f + h * r[6] / (3.0f * rho)) * rho * rho), r[12], 1.0f / h);
                }
            }
            __syncwarp();
            const uint32_t ball = __ballot_sync(0xFFFFFFFFu, ok), n_ok = __popc(ball);
            if (cnt + n_ok > kTile) { flush(cnt); cnt = 0; }
            if (ok) {
                const uint32_t pos = cnt + __popc(ball & lt);
                sm.ta[pos] = a; sm.tb[pos] = b; sm.tc[pos] = c;
            }
            cnt += n_ok;
        }
        if (cnt) flush(cnt);
        // results through shared memory so the 20-byte records leave as coalesced 16-byte stores
        if (valid) {
            float* o = sm.raw + 5 * lane;
            o[0] = ax; o[1] = ay; o[2] = az; o[3] = du; o[4] = vsig;
        }
        __syncwarp();
        const uint32_t nvec = (it.n_t * 5 + 3) >> 2;
        for (uint32_t v = lane; v < nvec; v += 32) reinterpret_cast<uint4*>(it.tout)[v] = reinterpret_cast<const uint4*>(sm.raw)[v];
        __syncwarp();
    }
}

template <class K>
int32_t loop_grid(K kernel, uint32_t n_items, uint32_t* grid) {
    int dev = 0, sms = 0, per_sm = 0;
    SPH_CUDA_TRY(cudaGetDevice(&dev));
    SPH_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    SPH_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kLoopWarps * 32, 0));
    *grid = min((n_items + kLoopWarps - 1) / kLoopWarps, (uint32_t)(sms * max(per_sm, 1)));
    return SPH_OK;
}

}  // namespace

int32_t launch_density(const sph_batch* b, const uint32_t* d_off_in, const uint32_t* d_off_out, const char* d_in, char* d_out, cudaStream_t st) {
    if (b->n_chunks == 0) return SPH_OK;
    static uint32_t full_grid = 0;
    if (!full_grid)
        if (int32_t rc = loop_grid(density_kernel, 0xFFFFFFFFu - kLoopWarps, &full_grid)) return rc;
    const uint32_t grid = min((b->n_chunks + kLoopWarps - 1) / kLoopWarps, full_grid);
    density_kernel<<<grid, kLoopWarps * 32, 0, st>>>(b->d_sides, b->d_chunk_side, b->d_chunk_src, d_off_in, d_off_out, d_in, d_out, b->n_chunks);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_force(const sph_batch* b, const uint32_t* d_off_in, const uint32_t* d_off_out, const char* d_in, char* d_out,
                     const sph_params& prm, cudaStream_t st) {
    if (b->n_chunks == 0) return SPH_OK;
    static uint32_t full_grid = 0;
    if (!full_grid)
        if (int32_t rc = loop_grid(force_kernel, 0xFFFFFFFFu - kLoopWarps, &full_grid)) return rc;
    const uint32_t grid = min((b->n_chunks + kLoopWarps - 1) / kLoopWarps, full_grid);
    force_kernel<<<grid, kLoopWarps * 32, 0, st>>>(b->d_sides, b->d_chunk_side, b->d_chunk_src, d_off_in, d_off_out, d_in, d_out,
                                                   b->n_chunks, prm.alpha, prm.beta);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
