// DENSITY and FORCE interaction loops over cell / cell-pair tasks.
//
// Nothing here is a dense contraction (a few percent of the candidate pairs are neighbours and the per-pair
// work is a distance test), so this is plain FP32 ALU work, not tensor-core work.
//
// Work item = (32 target particles of one block) x (the block they gather from: the task's other side, or the
// block itself for a self task); one 16-byte item descriptor, built with the batch.  One warp per item, warps
// never wait for one another (no __syncthreads):
//   (a) the 32 target records are staged through shared memory with coalesced 16-byte loads; the warp reduces
//       their bounding box and largest h with REDUX (integer min / max on an order-preserving image of the floats);
//   (b) the source block is streamed 32 records at a time the same way; a source outside the targets' reach box
//       (box grown by 2 h_max, for the force loop by max(2 h_max, 2 h_j)) cannot be anybody's neighbour and is
//       dropped; the others are compacted (ballot + popc) into a 64-entry tile;
//   (c) phase 1, a branch-free FILTER on two sources per instruction (fma.rn.f32x2 / add.rn.f32x2):
//       t = |s|^2 - 2 x_i.s + (|x_i|^2 - (2h)^2 - eps) = r^2 - (2h)^2 - eps, four packed operations per source pair;
//       the sign bit of t is funnel-shifted straight into a per-lane hit mask (one SHF per source).  eps covers the
//       rounding of the expanded form, so the mask is a superset of the neighbours;
//   (d) phase 2: every lane walks the set bits of its mask in source order, recomputes r^2 = |x_i - s|^2 exactly as
//       the definition does, applies the exact cut-off and evaluates the kernel terms.
// Sums are accumulated per lane in tile order = source order, so results are bit-reproducible run to run.
#include "internal.h"

namespace sph {

namespace {

constexpr int kLoopWarps = 4;
constexpr int kTile = 64;                  // compacted sources per flush = bits in the per-lane hit mask (2 x 32)
constexpr float kInvPi = 0.318309886183790671538f;
constexpr float kNever = 1.0e30f;          // |s|^2 of a tile pad entry / threshold of an idle lane: never a hit
constexpr float kReachSlack = 1.0f + 1.0e-4f;   // the reach box is a superset test; keep it clear of f32 rounding
constexpr float kFilterEps = 4.0e-6f;      // x (largest |coordinate|)^2 summed over the axes: bounds the rounding of the
                                           // expanded form (about 18 roundings of 2^-24 relative to that scale)
constexpr uint32_t kFull = 0xFFFFFFFFu;

// order-preserving image of a float in the signed integers, so that REDUX.MIN / REDUX.MAX reduce floats
__device__ __forceinline__ int ord(float f) { const int k = __float_as_int(f); return k ^ ((k >> 31) & 0x7FFFFFFF); }
__device__ __forceinline__ float unord(int k) { return __int_as_float(k ^ ((k >> 31) & 0x7FFFFFFF)); }
__device__ __forceinline__ float warp_min(float v, bool valid) { return unord(__reduce_min_sync(kFull, valid ? ord(v) : 0x7FFFFFFF)); }
__device__ __forceinline__ float warp_max(float v, bool valid) { return unord(__reduce_max_sync(kFull, valid ? ord(v) : (int)0x80000000)); }
__device__ __forceinline__ float warp_max_pos(float v) { return __uint_as_float(__reduce_max_sync(kFull, __float_as_uint(v))); }   // v >= 0

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
// packed pairs of f32 (sm_100: FADD2 / FFMA2, two sources per instruction)
__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long add2(unsigned long long a, unsigned long long b) {
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// n records of `words` 4-byte words, contiguous and 16-byte aligned in global memory -> raw (shared), coalesced
__device__ __forceinline__ void stage_records(float* raw, const char* g, uint32_t n, uint32_t words, uint32_t lane) {
    const uint32_t nvec = (n * words + 3) >> 2;   // a last partial vector reads into the block's pad bytes
    for (uint32_t v = lane; v < nvec; v += 32) reinterpret_cast<uint4*>(raw)[v] = __ldg(reinterpret_cast<const uint4*>(g) + v);
}

// cubic spline (M4), q = r/h in [0, 2]: value and derivative
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

// The filter's view of the tile: sources two by two, {x0, x1, y0, y1} and {z0, z1, |s0|^2, |s1|^2}.
struct FilterTile {
    float4 a[kTile / 2];
    float4 b[kTile / 2];
};
__device__ __forceinline__ void filter_put(FilterTile& f, uint32_t pos, float x, float y, float z, float s2) {
    float* a = reinterpret_cast<float*>(&f.a[pos >> 1]) + (pos & 1);
    float* b = reinterpret_cast<float*>(&f.b[pos >> 1]) + (pos & 1);
    a[0] = x; a[2] = y; b[0] = z; b[2] = s2;
}

// Phase 1 over the first `cnt` tile entries: bit (31 - j) of m0 = "source j may be a neighbour" (j < 32), m1 likewise
// for sources 32..63.  mx2, my2, mz2 = (-2 x_i) twice; nt2 = (|x_i|^2 - cut^2 - eps) twice.
__device__ __forceinline__ void filter_masks(FilterTile& f, uint32_t cnt, uint32_t lane, unsigned long long mx2, unsigned long long my2,
                                             unsigned long long mz2, unsigned long long nt2, uint32_t* m0_out, uint32_t* m1_out) {
    const uint32_t n4 = (cnt + 3) & ~3u;
    if (lane < n4 - cnt) filter_put(f, cnt + lane, 0.f, 0.f, 0.f, kNever);
    __syncwarp();
    const uint32_t np = n4 >> 1, np0 = min(np, 16u);
    uint32_t m0 = 0, m1 = 0;
    auto test2 = [&](uint32_t p, uint32_t& m) {
        const ulonglong2 a = *reinterpret_cast<const ulonglong2*>(&f.a[p]);
        const ulonglong2 b = *reinterpret_cast<const ulonglong2*>(&f.b[p]);
        unsigned long long t = add2(b.y, nt2);
        t = fma2(mz2, b.x, t);
        t = fma2(my2, a.y, t);
        t = fma2(mx2, a.x, t);
        uint32_t lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(t));
        m = __funnelshift_l(lo, m, 1);      // (m << 1) | sign(t_lo)
        m = __funnelshift_l(hi, m, 1);
    };
    for (uint32_t p = 0; p < np0; p += 2) { test2(p, m0); test2(p + 1, m0); }
    m0 <<= 32 - 2 * np0;
    if (np > 16) {
        for (uint32_t p = 16; p < np; p += 2) { test2(p, m1); test2(p + 1, m1); }
        m1 <<= 32 - 2 * (np - 16);
    }
    *m0_out = m0;
    *m1_out = m1;
}

// next candidate of a lane in source order; false when the lane has none left
__device__ __forceinline__ bool next_hit(uint32_t& m0, uint32_t& m1, uint32_t* j) {
    const bool first = m0 != 0;
    const uint32_t m = first ? m0 : m1;
    if (m == 0) return false;
    const uint32_t z = __clz(m), bit = 0x80000000u >> z;
    if (first) m0 ^= bit; else m1 ^= bit;
    *j = z + (first ? 0u : 32u);
    return true;
}

// ------------------------------------------------------------------------------------------------- density

struct DensityWarpSmem {
    FilterTile f;
    float4 tile[kTile];      // x, y, z, m of the compacted sources
    float raw[32 * 5];       // staging of 32 DENSITY_IN records: xr0 xr1 xr2 h m
};

__global__ void __launch_bounds__(kLoopWarps * 32)
density_kernel(const LoopItem* __restrict__ items, const char* __restrict__ in, char* __restrict__ out, uint32_t n_items) {
    __shared__ __align__(16) DensityWarpSmem s_all[kLoopWarps];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    DensityWarpSmem& sm = s_all[warp];
    const uint32_t lt = lanemask_lt();

    for (uint32_t item = blockIdx.x * kLoopWarps + warp; item < n_items; item += gridDim.x * kLoopWarps) {
        const uint4 iw = __ldg(reinterpret_cast<const uint4*>(items) + item);
        const uint32_t n_t = iw.w & 63u, n_s = iw.w >> 6;
        const char* sin = in + (uint64_t)iw.y * 128;
        stage_records(sm.raw, in + (uint64_t)iw.x * 128, n_t, 5, lane);
        __syncwarp();
        const bool valid = lane < n_t;
        const float xi = valid ? sm.raw[5 * lane] : 0.f, yi = valid ? sm.raw[5 * lane + 1] : 0.f, zi = valid ? sm.raw[5 * lane + 2] : 0.f;
        const float hi = valid ? sm.raw[5 * lane + 3] : 0.f;
        __syncwarp();
        const float hc2 = 4.0f * hi * hi, inv_h = valid ? 1.0f / hi : 0.f;
        const float reach = 2.0f * warp_max_pos(hi) * kReachSlack;
        const float lox = warp_min(xi, valid) - reach, hix = warp_max(xi, valid) + reach;
        const float loy = warp_min(yi, valid) - reach, hiy = warp_max(yi, valid) + reach;
        const float loz = warp_min(zi, valid) - reach, hiz = warp_max(zi, valid) + reach;
        const float bx = fmaxf(fabsf(lox), fabsf(hix)), by = fmaxf(fabsf(loy), fabsf(hiy)), bz = fmaxf(fabsf(loz), fabsf(hiz));
        const float eps = kFilterEps * fmaf(bx, bx, fmaf(by, by, bz * bz));
        const float nt = valid ? fmaf(xi, xi, fmaf(yi, yi, zi * zi)) - hc2 - eps : kNever;
        const unsigned long long mx2 = pack2(-2.0f * xi, -2.0f * xi), my2 = pack2(-2.0f * yi, -2.0f * yi), mz2 = pack2(-2.0f * zi, -2.0f * zi);
        const unsigned long long nt2 = pack2(nt, nt);
        float s_mw = 0.f, s_mg = 0.f, s_w = 0.f, s_g = 0.f;     // sums of m w, m (3w + q w'), w, (3w + q w')

        auto flush = [&](uint32_t cnt) {
            uint32_t m0, m1, j;
            filter_masks(sm.f, cnt, lane, mx2, my2, mz2, nt2, &m0, &m1);
            while (next_hit(m0, m1, &j)) {
                const float4 s = sm.tile[j];
                const float dx = xi - s.x, dy = yi - s.y, dz = zi - s.z;
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                // a filter false positive has r2 >= (2h)^2: q clamps to 2 where w = w' = 0 exactly
                const float q = fminf(sqrt_approx(r2) * inv_h, 2.0f);
                float w, dw;
                spline(q, &w, &dw);
                const float g = fmaf(q, dw, 3.0f * w);
                s_mw = fmaf(s.w, w, s_mw); s_mg = fmaf(s.w, g, s_mg);
                s_w += w; s_g += g;
            }
            __syncwarp();
        };

        uint32_t cnt = 0;
        for (uint32_t j0 = 0; j0 < n_s; j0 += 32) {
            const uint32_t nj = min(32u, n_s - j0);
            stage_records(sm.raw, sin + (uint64_t)j0 * 20, nj, 5, lane);
            __syncwarp();
            float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
            bool ok = false;
            if (lane < nj) {
                s = make_float4(sm.raw[5 * lane], sm.raw[5 * lane + 1], sm.raw[5 * lane + 2], sm.raw[5 * lane + 4]);
                ok = s.x > lox && s.x < hix && s.y > loy && s.y < hiy && s.z > loz && s.z < hiz;
            }
            __syncwarp();
            const uint32_t ball = __ballot_sync(kFull, ok), c = __popc(ball);
            if (cnt + c > kTile) { flush(cnt); cnt = 0; }
            if (ok) {
                const uint32_t pos = cnt + __popc(ball & lt);
                sm.tile[pos] = s;
                filter_put(sm.f, pos, s.x, s.y, s.z, fmaf(s.x, s.x, fmaf(s.y, s.y, s.z * s.z)));
            }
            cnt += c;
        }
        if (cnt) flush(cnt);
        if (valid) {
            const float n3 = kInvPi * inv_h * inv_h * inv_h, n4 = n3 * inv_h;
            reinterpret_cast<float4*>(out + (uint64_t)iw.z * 128)[lane] = make_float4(s_mw * n3, -s_mg * n4, s_w * n3, -s_g * n4);
        }
    }
}

// ------------------------------------------------------------------------------------------------- force

struct ForceWarpSmem {
    FilterTile f;
    float4 ta[kTile];        // x, y, z, 4 h^2
    float4 tb[kTile];        // vx, vy, vz, m
    float4 tc[kTile];        // rho, A = P / (Omega rho^2), c_s, 1/h
    float raw[32 * 13];      // staging of 32 FORCE_IN records: xr0 xr1 xr2 h m rho rho_dh v0 v1 v2 u P cs (and of the 32 results)
};

__global__ void __launch_bounds__(kLoopWarps * 32)
force_kernel(const LoopItem* __restrict__ items, const char* __restrict__ in, char* __restrict__ out, uint32_t n_items, float alpha, float beta) {
    __shared__ __align__(16) ForceWarpSmem s_all[kLoopWarps];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ForceWarpSmem& sm = s_all[warp];
    const uint32_t lt = lanemask_lt();

    for (uint32_t item = blockIdx.x * kLoopWarps + warp; item < n_items; item += gridDim.x * kLoopWarps) {
        const uint4 iw = __ldg(reinterpret_cast<const uint4*>(items) + item);
        const uint32_t n_t = iw.w & 63u, n_s = iw.w >> 6;
        const char* sin = in + (uint64_t)iw.y * 128;
        stage_records(sm.raw, in + (uint64_t)iw.x * 128, n_t, 13, lane);
        __syncwarp();
        const bool valid = lane < n_t;
        float xi = 0.f, yi = 0.f, zi = 0.f, hi = 0.f, rhoi = 1.f, rho_dhi = 0.f, vxi = 0.f, vyi = 0.f, vzi = 0.f, Pi = 0.f, ci = 0.f;
        if (valid) {
            const float* r = sm.raw + 13 * lane;
            xi = r[0]; yi = r[1]; zi = r[2]; hi = r[3]; rhoi = r[5]; rho_dhi = r[6]; vxi = r[7]; vyi = r[8]; vzi = r[9]; Pi = r[11]; ci = r[12];
        }
        __syncwarp();
        const float hc2i = 4.0f * hi * hi, inv_hi = valid ? 1.0f / hi : 0.f;
        const float n4i = kInvPi * (inv_hi * inv_hi) * (inv_hi * inv_hi);
        const float Ai = Pi / ((1.0f + hi * rho_dhi / (3.0f * rhoi)) * rhoi * rhoi);
        const float reach_t = 2.0f * warp_max_pos(hi);
        const float lox = warp_min(xi, valid), hix = warp_max(xi, valid);
        const float loy = warp_min(yi, valid), hiy = warp_max(yi, valid);
        const float loz = warp_min(zi, valid), hiz = warp_max(zi, valid);
        const float ri2 = fmaf(xi, xi, fmaf(yi, yi, zi * zi));
        const float ri2_max = warp_max_pos(ri2);
        const unsigned long long mx2 = pack2(-2.0f * xi, -2.0f * xi), my2 = pack2(-2.0f * yi, -2.0f * yi), mz2 = pack2(-2.0f * zi, -2.0f * zi);
        float ax = 0.f, ay = 0.f, az = 0.f, du = 0.f, vsig = 0.f;
        float tile_hc2 = 0.f, tile_b2 = 0.f;      // over the tile being filled: largest (2 h_j)^2, largest |s|^2 (warp-uniform)

        auto flush = [&](uint32_t cnt) {
            // filter cut-off of a lane: max((2 h_i)^2, largest (2 h_j)^2 in the tile) -- a superset of max(2h_i, 2h_j) per pair
            const float cut2 = fmaxf(hc2i, tile_hc2);
            const float eps = kFilterEps * fmaf(3.0f, fmaxf(tile_b2, ri2_max), cut2);
            const float nt = valid ? ri2 - cut2 - eps : kNever;
            uint32_t m0, m1, j;
            filter_masks(sm.f, cnt, lane, mx2, my2, mz2, pack2(nt, nt), &m0, &m1);
            while (next_hit(m0, m1, &j)) {
                const float4 a = sm.ta[j];
                const float dx = xi - a.x, dy = yi - a.y, dz = zi - a.z;
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                if (!(r2 < fmaxf(hc2i, a.w) && r2 > 0.f)) continue;      // the exact cut-off; r = 0 is the particle itself
                const float4 b = sm.tb[j], c = sm.tc[j];
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
            }
            tile_hc2 = 0.f; tile_b2 = 0.f;
            __syncwarp();
        };

        uint32_t cnt = 0;
        for (uint32_t j0 = 0; j0 < n_s; j0 += 32) {
            const uint32_t nj = min(32u, n_s - j0);
            stage_records(sm.raw, sin + (uint64_t)j0 * 52, nj, 13, lane);
            __syncwarp();
            float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a, c = a;
            float s2 = 0.f;
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
                    s2 = fmaf(a.x, a.x, fmaf(a.y, a.y, a.z * a.z));
                }
            }
            __syncwarp();
            const uint32_t ball = __ballot_sync(kFull, ok), n_ok = __popc(ball);
            if (cnt + n_ok > kTile) { flush(cnt); cnt = 0; }
            if (ok) {
                const uint32_t pos = cnt + __popc(ball & lt);
                sm.ta[pos] = a; sm.tb[pos] = b; sm.tc[pos] = c;
                filter_put(sm.f, pos, a.x, a.y, a.z, s2);
            }
            tile_hc2 = fmaxf(tile_hc2, warp_max_pos(ok ? a.w : 0.f));
            tile_b2 = fmaxf(tile_b2, warp_max_pos(s2));
            cnt += n_ok;
        }
        if (cnt) flush(cnt);
        // results through shared memory so the 20-byte records leave as coalesced 16-byte stores
        if (valid) {
            float* o = sm.raw + 5 * lane;
            o[0] = ax; o[1] = ay; o[2] = az; o[3] = du; o[4] = vsig;
        }
        __syncwarp();
        const uint32_t nvec = (n_t * 5 + 3) >> 2;
        char* tout = out + (uint64_t)iw.z * 128;
        for (uint32_t v = lane; v < nvec; v += 32) reinterpret_cast<uint4*>(tout)[v] = reinterpret_cast<const uint4*>(sm.raw)[v];
        __syncwarp();
    }
}

template <class K>
int32_t loop_grid(K kernel, uint32_t* grid) {
    int dev = 0, sms = 0, per_sm = 0;
    SPH_CUDA_TRY(cudaGetDevice(&dev));
    SPH_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    SPH_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kLoopWarps * 32, 0));
    *grid = (uint32_t)(sms * max(per_sm, 1));
    return SPH_OK;
}

}  // namespace

int32_t launch_density(const sph_batch* b, const char* d_in, char* d_out, cudaStream_t st) {
    if (b->n_chunks == 0) return SPH_OK;
    static uint32_t full_grid = 0;
    if (!full_grid)
        if (int32_t rc = loop_grid(density_kernel, &full_grid)) return rc;
    const uint32_t grid = min((b->n_chunks + kLoopWarps - 1) / kLoopWarps, full_grid);
    density_kernel<<<grid, kLoopWarps * 32, 0, st>>>(b->d_items_density, d_in, d_out, b->n_chunks);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_force(const sph_batch* b, const char* d_in, char* d_out, const sph_params& prm, cudaStream_t st) {
    if (b->n_chunks == 0) return SPH_OK;
    static uint32_t full_grid = 0;
    if (!full_grid)
        if (int32_t rc = loop_grid(force_kernel, &full_grid)) return rc;
    const uint32_t grid = min((b->n_chunks + kLoopWarps - 1) / kLoopWarps, full_grid);
    force_kernel<<<grid, kLoopWarps * 32, 0, st>>>(b->d_items_force, d_in, d_out, b->n_chunks, prm.alpha, prm.beta);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
