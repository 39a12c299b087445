// DENSITY and FORCE interaction loops over cell / cell-pair tasks.
//
// Nothing here is a dense contraction (a few percent of the candidate pairs are neighbours and the per-pair
// work is a distance test), so this is plain FP32 ALU work, not tensor-core work.
//
// Work item = (up to 64 target particles of one block, two per lane: A = lane, B = lane + 32) x (the block they
// gather from: the task's other side, or the block itself for a self task); one 16-byte item descriptor, built
// with the batch.  One warp per item, warps never wait for one another (no __syncthreads):
//   (a) records travel global -> shared memory as coalesced 16-byte cp.async copies, one step AHEAD of their use:
//       while a round of 32 source records is processed the next round (or the next item's targets and first
//       round) is already in flight;
//   (b) the warp reduces the targets' bounding box and largest h with REDUX (integer min / max on an
//       order-preserving image of the floats); a source outside the reach box (box grown by 2 h_max, for the
//       force loop by max(2 h_max, 2 h_j)) cannot be anybody's neighbour and is dropped; the others are compacted
//       (ballot + popc) into a 64-entry tile;
//   (c) phase 1, a branch-free FILTER on two sources per instruction (fma.rn.f32x2 / add.rn.f32x2):
//       t = |s|^2 - 2 x_i.s + (|x_i|^2 - (2h)^2 - eps) = r^2 - (2h)^2 - eps, four packed operations per source pair
//       and target; the sign bit of t is funnel-shifted straight into a per-target hit mask (one SHF per source).
//       eps covers the rounding of the expanded form, so the mask is a superset of the neighbours;
//   (d) phase 2: every lane walks the set bits of its two masks in source order, one hit of target A and one of
//       target B per iteration, the pair evaluated with packed f32x2 arithmetic (a target that has run out of
//       hits is fed a far-away dummy source whose contribution is exactly zero).  r^2 = |x_i - s|^2 is recomputed
//       exactly as the definition does and the exact cut-off applied.
// Sums are accumulated per target in tile order = source order, so results are bit-reproducible run to run.
#include "internal.h"

namespace sph {

namespace {

typedef unsigned long long u64;            // a pair of f32 (lo = target A, hi = target B)

constexpr int kLoopWarps = 4;
constexpr int kTile = 64;                  // compacted sources per flush: two halves of 32, one mask word each per target
constexpr int kHalf = 33;                  // tile entries per half: 32 sources + the dummy (where __clz(0) = 32 points)
constexpr float kInvPi = 0.318309886183790671538f;
constexpr float kNever = 1.0e30f;          // |s|^2 of a filter pad entry / threshold of an idle target: never a hit
constexpr float kFar = 1.0e15f;            // coordinates of the dummy source (r^2 = 3e30 stays finite)
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
__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ uint32_t lanemask_lt() {
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}
__device__ __forceinline__ uint32_t shr_clamp(uint32_t v, uint32_t n) {   // PTX shr clamps the amount: n >= 32 gives 0
    uint32_t r;
    asm("shr.b32 %0, %1, %2;" : "=r"(r) : "r"(v), "r"(n));
    return r;
}
// packed pairs of f32 (sm_100: FADD2 / FMUL2 / FFMA2, two values per instruction)
__device__ __forceinline__ u64 pack2(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 dup2(float v) { return pack2(v, v); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 sub2(u64 a, u64 b) {
    u64 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// n (<= MAXREC) records of WORDS 4-byte words, contiguous and 16-byte aligned in global memory -> shared, coalesced and asynchronous.
// A last partial vector reads into the block's pad bytes.
template <int WORDS, int MAXREC>
__device__ __forceinline__ void fetch_records(float* dst, const char* g, uint32_t n, uint32_t lane) {
    const uint32_t nvec = (n * WORDS + 3) >> 2;
    constexpr int NV = (MAXREC * WORDS / 4 + 31) / 32;
#pragma unroll
    for (int it = 0; it < NV; ++it) {
        const uint32_t v = lane + 32 * it;
        if (v < nvec) cp_async16(dst + 4 * v, g + 16 * (size_t)v);
    }
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

// The filter constants of one target: (-2 x_i) twice per axis and (|x_i|^2 - cut^2 - eps) twice.
struct FilterTarget {
    u64 mx2, my2, mz2, nt2;
};
__device__ __forceinline__ FilterTarget filter_target(float x, float y, float z, float nt) {
    return FilterTarget{dup2(-2.0f * x), dup2(-2.0f * y), dup2(-2.0f * z), dup2(nt)};
}

// Phase 1 over the first `cnt` tile entries for the lane's two targets: bit (31 - j) of m[0] = "source j may be a
// neighbour of target A" (j < 32), m[1] likewise for sources 32..63; m[2], m[3] for target B.
__device__ __forceinline__ void filter_masks(FilterTile& f, uint32_t cnt, uint32_t lane, const FilterTarget& A, const FilterTarget& B, uint32_t (&m)[4]) {
    const uint32_t n4 = (cnt + 3) & ~3u;
    if (lane < n4 - cnt) filter_put(f, cnt + lane, 0.f, 0.f, 0.f, kNever);
    __syncwarp();
    const uint32_t np = n4 >> 1, np0 = min(np, 16u);
    uint32_t a0 = 0, a1 = 0, b0 = 0, b1 = 0;
    auto test2 = [&](uint32_t p, uint32_t& ma, uint32_t& mb) {
        const ulonglong2 a = *reinterpret_cast<const ulonglong2*>(&f.a[p]);
        const ulonglong2 b = *reinterpret_cast<const ulonglong2*>(&f.b[p]);
        const u64 ta = fma2(A.mx2, a.x, fma2(A.my2, a.y, fma2(A.mz2, b.x, add2(b.y, A.nt2))));
        const u64 tb = fma2(B.mx2, a.x, fma2(B.my2, a.y, fma2(B.mz2, b.x, add2(b.y, B.nt2))));
        uint32_t lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(ta));
        ma = __funnelshift_l(lo, ma, 1);      // (m << 1) | sign(t_lo)
        ma = __funnelshift_l(hi, ma, 1);
        asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(tb));
        mb = __funnelshift_l(lo, mb, 1);
        mb = __funnelshift_l(hi, mb, 1);
    };
    for (uint32_t p = 0; p < np0; p += 2) { test2(p, a0, b0); test2(p + 1, a0, b0); }
    a0 <<= 32 - 2 * np0; b0 <<= 32 - 2 * np0;
    if (np > 16) {
        for (uint32_t p = 16; p < np; p += 2) { test2(p, a1, b1); test2(p + 1, a1, b1); }
        a1 <<= 32 - 2 * (np - 16); b1 <<= 32 - 2 * (np - 16);
    }
    m[0] = a0; m[1] = a1; m[2] = b0; m[3] = b1;
}

// next hit of each of the two targets in one half of the tile (32 = the dummy when a target has none left)
__device__ __forceinline__ void next_hits(uint32_t& ma, uint32_t& mb, uint32_t* ja, uint32_t* jb) {
    *ja = __clz(ma); *jb = __clz(mb);
    ma &= ~shr_clamp(0x80000000u, *ja);
    mb &= ~shr_clamp(0x80000000u, *jb);
}

// the lane's two targets as a pair: value of A in the low half, of B in the high half
__device__ __forceinline__ u64 load2(const float* rec, uint32_t stride, uint32_t word, uint32_t lane, bool vA, bool vB, float idle) {
    return pack2(vA ? rec[stride * lane + word] : idle, vB ? rec[stride * (lane + 32) + word] : idle);
}

// ------------------------------------------------------------------------------------------------- density

struct DensityWarpSmem {
    FilterTile f;
    float4 tile[2 * kHalf];  // x, y, z, m of the compacted sources; entries 32 and 65 are the dummy
    float tgt[64 * 5];       // landing area of an item's 64 DENSITY_IN records: xr0 xr1 xr2 h m
    float src[2][32 * 5];    // landing areas of the source rounds (double-buffered)
};

__global__ void __launch_bounds__(kLoopWarps * 32)
density_kernel(const LoopItem* __restrict__ items, const char* __restrict__ in, char* __restrict__ out, uint32_t n_items) {
    __shared__ __align__(16) DensityWarpSmem s_all[kLoopWarps];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    DensityWarpSmem& sm = s_all[warp];
    const uint32_t lt = lanemask_lt();
    const uint32_t step = gridDim.x * kLoopWarps;
    uint32_t item = blockIdx.x * kLoopWarps + warp;
    if (item >= n_items) return;
    if (lane < 2) sm.tile[lane * kHalf + 32] = make_float4(kFar, kFar, kFar, 0.f);
    const u64 kTwo = dup2(2.0f), kThree = dup2(3.0f), kQuarter = dup2(0.25f), kM075 = dup2(-0.75f);

    uint4 iw = __ldg(reinterpret_cast<const uint4*>(items) + item);
    fetch_records<5, 64>(sm.tgt, in + (uint64_t)iw.x * 128, iw.w & 127u, lane);
    fetch_records<5, 32>(sm.src[0], in + (uint64_t)iw.y * 128, min(32u, iw.w >> 7), lane);
    uint32_t buf = 0;

    for (; item < n_items; item += step) {
        const uint32_t n_t = iw.w & 127u, n_s = iw.w >> 7;
        const char* sin = in + (uint64_t)iw.y * 128;
        char* tout = out + (uint64_t)iw.z * 128;
        const bool has_next = item + step < n_items;
        uint4 iw_next = iw;
        if (has_next) iw_next = __ldg(reinterpret_cast<const uint4*>(items) + item + step);
        cp_async_wait_all();          // this item's targets and first source round
        __syncwarp();
        const bool vA = lane < n_t, vB = lane + 32 < n_t;
        const u64 x2 = load2(sm.tgt, 5, 0, lane, vA, vB, 0.f), y2 = load2(sm.tgt, 5, 1, lane, vA, vB, 0.f), z2 = load2(sm.tgt, 5, 2, lane, vA, vB, 0.f);
        float xA, xB, yA, yB, zA, zB;
        unpack2(x2, xA, xB); unpack2(y2, yA, yB); unpack2(z2, zA, zB);
        const float hA = vA ? sm.tgt[5 * lane + 3] : 0.f, hB = vB ? sm.tgt[5 * (lane + 32) + 3] : 0.f;
        __syncwarp();                 // sm.tgt may now receive the next item's targets
        const float inv_hA = vA ? 1.0f / hA : 0.f, inv_hB = vB ? 1.0f / hB : 0.f;
        const float reach = 2.0f * warp_max_pos(fmaxf(hA, hB)) * kReachSlack;
        const float lox = warp_min(vB ? fminf(xA, xB) : xA, vA) - reach, hix = warp_max(vB ? fmaxf(xA, xB) : xA, vA) + reach;
        const float loy = warp_min(vB ? fminf(yA, yB) : yA, vA) - reach, hiy = warp_max(vB ? fmaxf(yA, yB) : yA, vA) + reach;
        const float loz = warp_min(vB ? fminf(zA, zB) : zA, vA) - reach, hiz = warp_max(vB ? fmaxf(zA, zB) : zA, vA) + reach;
        const float bx = fmaxf(fabsf(lox), fabsf(hix)), by = fmaxf(fabsf(loy), fabsf(hiy)), bz = fmaxf(fabsf(loz), fabsf(hiz));
        const float eps = kFilterEps * fmaf(bx, bx, fmaf(by, by, bz * bz));
        const FilterTarget fA = filter_target(xA, yA, zA, vA ? fmaf(xA, xA, fmaf(yA, yA, zA * zA)) - 4.0f * hA * hA - eps : kNever);
        const FilterTarget fB = filter_target(xB, yB, zB, vB ? fmaf(xB, xB, fmaf(yB, yB, zB * zB)) - 4.0f * hB * hB - eps : kNever);
        u64 s_mw = 0, s_mg = 0, s_w = 0, s_g = 0;     // sums of m w, m (3w + q w'), w, (3w + q w') for (A, B)

        // phase 2 over one half of the tile
        auto hits = [&](uint32_t ma, uint32_t mb, const float4* half) {
            while ((ma | mb) != 0) {
                uint32_t ja, jb;
                next_hits(ma, mb, &ja, &jb);
                const float4 a = half[ja], b = half[jb];
                const u64 dx = sub2(x2, pack2(a.x, b.x)), dy = sub2(y2, pack2(a.y, b.y)), dz = sub2(z2, pack2(a.z, b.z));
                const u64 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
                float r2a, r2b;
                unpack2(r2, r2a, r2b);
                // a filter false positive has r2 >= (2h)^2: q clamps to 2 where w = w' = 0 exactly (and so does the dummy)
                const float qa = fminf(sqrt_approx(r2a) * inv_hA, 2.0f), qb = fminf(sqrt_approx(r2b) * inv_hB, 2.0f);
                const u64 q = pack2(qa, qb), u = pack2(fminf(qa - 1.0f, 0.f), fminf(qb - 1.0f, 0.f));   // u = -(1 - q)+
                const u64 t = sub2(kTwo, q);                                                                // t = (2 - q)+
                const u64 tt = mul2(t, t), uu = mul2(u, u);
                const u64 w = fma2(mul2(kQuarter, t), tt, mul2(u, uu));      // 0.25 t^3 - (1 - q)+^3
                const u64 dw = fma2(kThree, uu, mul2(kM075, tt));            // -0.75 t^2 + 3 (1 - q)+^2
                const u64 g = fma2(q, dw, mul2(kThree, w));
                const u64 m = pack2(a.w, b.w);
                s_mw = fma2(m, w, s_mw); s_mg = fma2(m, g, s_mg);
                s_w = add2(s_w, w); s_g = add2(s_g, g);
            }
        };
        auto flush = [&](uint32_t cnt) {
            uint32_t m[4];
            filter_masks(sm.f, cnt, lane, fA, fB, m);
            hits(m[0], m[2], sm.tile);
            if (cnt > 32) hits(m[1], m[3], sm.tile + kHalf);
            __syncwarp();
        };

        uint32_t cnt = 0;
        const uint32_t n_rounds = max(1u, (n_s + 31) >> 5);
        for (uint32_t r = 0; r < n_rounds; ++r) {
            const uint32_t j0 = 32 * r, nj = min(32u, n_s - j0);
            if (r > 0) { cp_async_wait_all(); __syncwarp(); }
            // one step ahead: the next round of this item, or the next item's targets and first round
            if (r + 1 < n_rounds) {
                fetch_records<5, 32>(sm.src[buf ^ 1], sin + (uint64_t)(j0 + 32) * 20, min(32u, n_s - j0 - 32), lane);
            } else if (has_next) {
                fetch_records<5, 64>(sm.tgt, in + (uint64_t)iw_next.x * 128, iw_next.w & 127u, lane);
                fetch_records<5, 32>(sm.src[buf ^ 1], in + (uint64_t)iw_next.y * 128, min(32u, iw_next.w >> 7), lane);
            }
            float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
            bool ok = false;
            if (lane < nj) {
                const float* rec = sm.src[buf] + 5 * lane;
                s = make_float4(rec[0], rec[1], rec[2], rec[4]);
                ok = s.x > lox && s.x < hix && s.y > loy && s.y < hiy && s.z > loz && s.z < hiz;
            }
            const uint32_t ball = __ballot_sync(kFull, ok), c = __popc(ball);
            if (cnt + c > kTile) { flush(cnt); cnt = 0; }
            if (ok) {
                const uint32_t pos = cnt + __popc(ball & lt);
                sm.tile[pos + (pos >> 5)] = s;        // half * 33 + index in the half
                filter_put(sm.f, pos, s.x, s.y, s.z, fmaf(s.x, s.x, fmaf(s.y, s.y, s.z * s.z)));
            }
            cnt += c;
            buf ^= 1;
        }
        if (cnt) flush(cnt);
        float mwA, mwB, mgA, mgB, wA, wB, gA, gB;
        unpack2(s_mw, mwA, mwB); unpack2(s_mg, mgA, mgB); unpack2(s_w, wA, wB); unpack2(s_g, gA, gB);
        if (vA) {
            const float n3 = kInvPi * inv_hA * inv_hA * inv_hA, n4 = n3 * inv_hA;
            reinterpret_cast<float4*>(tout)[lane] = make_float4(mwA * n3, -mgA * n4, wA * n3, -gA * n4);
        }
        if (vB) {
            const float n3 = kInvPi * inv_hB * inv_hB * inv_hB, n4 = n3 * inv_hB;
            reinterpret_cast<float4*>(tout)[lane + 32] = make_float4(mwB * n3, -mgB * n4, wB * n3, -gB * n4);
        }
        iw = iw_next;
    }
}

// ------------------------------------------------------------------------------------------------- force

struct ForceWarpSmem {
    FilterTile f;
    float4 ta[2 * kHalf];    // x, y, z, 4 h^2           (entries 32 and 65: the dummy)
    float4 tb[2 * kHalf];    // vx, vy, vz, m
    float4 tc[2 * kHalf];    // rho, A = P / (Omega rho^2), c_s, 1/h
    float tgt[64 * 13];      // landing area of an item's 64 FORCE_IN records: xr0 xr1 xr2 h m rho rho_dh v0 v1 v2 u P cs
                             // (and, at the end of the item, of its 64 x 5 results)
    float src[2][32 * 13];   // landing areas of the source rounds (double-buffered)
};

// -0.75 (2 - q)+^2 + 3 (1 - q)+^2 = w'(q) of the cubic spline for a pair of q
__device__ __forceinline__ u64 spline_dw2(u64 q, u64 kTwo, u64 kOne, u64 kThree, u64 kM075) {
    float ta, tb, ua, ub;
    unpack2(sub2(kTwo, q), ta, tb);
    unpack2(sub2(kOne, q), ua, ub);
    const u64 t = pack2(fmaxf(ta, 0.f), fmaxf(tb, 0.f)), u = pack2(fmaxf(ua, 0.f), fmaxf(ub, 0.f));
    return fma2(kThree, mul2(u, u), mul2(kM075, mul2(t, t)));
}

__global__ void __launch_bounds__(kLoopWarps * 32)
force_kernel(const LoopItem* __restrict__ items, const char* __restrict__ in, char* __restrict__ out, uint32_t n_items, float alpha, float beta) {
    extern __shared__ __align__(16) unsigned char s_raw[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ForceWarpSmem& sm = reinterpret_cast<ForceWarpSmem*>(s_raw)[warp];
    const uint32_t lt = lanemask_lt();
    const uint32_t step = gridDim.x * kLoopWarps;
    uint32_t item = blockIdx.x * kLoopWarps + warp;
    if (item >= n_items) return;
    if (lane < 2) {
        sm.ta[lane * kHalf + 32] = make_float4(kFar, kFar, kFar, 0.f);
        sm.tb[lane * kHalf + 32] = make_float4(0.f, 0.f, 0.f, 0.f);
        sm.tc[lane * kHalf + 32] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    const u64 kTwo = dup2(2.0f), kOne = dup2(1.0f), kThree = dup2(3.0f), kM075 = dup2(-0.75f), kHalf2 = dup2(0.5f), kMHalf2 = dup2(-0.5f),
              kOneHalf2 = dup2(1.5f), kInvPi2 = dup2(kInvPi), kMBeta2 = dup2(-beta), kMAlpha2 = dup2(-alpha);

    uint4 iw = __ldg(reinterpret_cast<const uint4*>(items) + item);
    fetch_records<13, 64>(sm.tgt, in + (uint64_t)iw.x * 128, iw.w & 127u, lane);
    fetch_records<13, 32>(sm.src[0], in + (uint64_t)iw.y * 128, min(32u, iw.w >> 7), lane);
    uint32_t buf = 0;

    for (; item < n_items; item += step) {
        const uint32_t n_t = iw.w & 127u, n_s = iw.w >> 7;
        const char* sin = in + (uint64_t)iw.y * 128;
        char* tout = out + (uint64_t)iw.z * 128;
        const bool has_next = item + step < n_items;
        uint4 iw_next = iw;
        if (has_next) iw_next = __ldg(reinterpret_cast<const uint4*>(items) + item + step);
        cp_async_wait_all();          // this item's targets and first source round
        __syncwarp();
        const bool vA = lane < n_t, vB = lane + 32 < n_t;
        const u64 x2 = load2(sm.tgt, 13, 0, lane, vA, vB, 0.f), y2 = load2(sm.tgt, 13, 1, lane, vA, vB, 0.f), z2 = load2(sm.tgt, 13, 2, lane, vA, vB, 0.f);
        const u64 h2 = load2(sm.tgt, 13, 3, lane, vA, vB, 0.f), rho2 = load2(sm.tgt, 13, 5, lane, vA, vB, 1.f), rho_dh2 = load2(sm.tgt, 13, 6, lane, vA, vB, 0.f);
        const u64 vx2 = load2(sm.tgt, 13, 7, lane, vA, vB, 0.f), vy2 = load2(sm.tgt, 13, 8, lane, vA, vB, 0.f), vz2 = load2(sm.tgt, 13, 9, lane, vA, vB, 0.f);
        const u64 P2 = load2(sm.tgt, 13, 11, lane, vA, vB, 0.f), c2 = load2(sm.tgt, 13, 12, lane, vA, vB, 0.f);
        __syncwarp();                 // sm.tgt may now receive the next item's targets (it is parked until the last round)
        float xA, xB, yA, yB, zA, zB, hA, hB, rhoA, rhoB, rdA, rdB, PA, PB;
        unpack2(x2, xA, xB); unpack2(y2, yA, yB); unpack2(z2, zA, zB); unpack2(h2, hA, hB);
        unpack2(rho2, rhoA, rhoB); unpack2(rho_dh2, rdA, rdB); unpack2(P2, PA, PB);
        const float hc2A = 4.0f * hA * hA, hc2B = 4.0f * hB * hB;
        const float inv_hA = vA ? 1.0f / hA : 0.f, inv_hB = vB ? 1.0f / hB : 0.f;
        const u64 inv_h2 = pack2(inv_hA, inv_hB);
        const u64 n42 = pack2(kInvPi * (inv_hA * inv_hA) * (inv_hA * inv_hA), kInvPi * (inv_hB * inv_hB) * (inv_hB * inv_hB));
        const u64 A2 = pack2(PA / ((1.0f + hA * rdA / (3.0f * rhoA)) * rhoA * rhoA), PB / ((1.0f + hB * rdB / (3.0f * rhoB)) * rhoB * rhoB));
        const float reach_t = 2.0f * warp_max_pos(fmaxf(hA, hB));
        const float lox = warp_min(vB ? fminf(xA, xB) : xA, vA), hix = warp_max(vB ? fmaxf(xA, xB) : xA, vA);
        const float loy = warp_min(vB ? fminf(yA, yB) : yA, vA), hiy = warp_max(vB ? fmaxf(yA, yB) : yA, vA);
        const float loz = warp_min(vB ? fminf(zA, zB) : zA, vA), hiz = warp_max(vB ? fmaxf(zA, zB) : zA, vA);
        const float ri2A = fmaf(xA, xA, fmaf(yA, yA, zA * zA)), ri2B = fmaf(xB, xB, fmaf(yB, yB, zB * zB));
        const float ri2_max = warp_max_pos(fmaxf(ri2A, ri2B));
        u64 ax = 0, ay = 0, az = 0, du = 0;
        float vsigA = 0.f, vsigB = 0.f;
        float tile_hc2 = 0.f, tile_b2 = 0.f;      // over the tile being filled: largest (2 h_j)^2, largest |s|^2 (warp-uniform)

        // phase 2 over one half of the tile.  e = x_j - x_i and v_j - v_i are used (both signs flipped): (v_i - v_j).(x_i - x_j)
        // is the same number and a_i += -m (..) (x_i - x_j) / r becomes one fma with e.
        auto hits = [&](uint32_t ma, uint32_t mb, uint32_t base) {
            while ((ma | mb) != 0) {
                uint32_t ja, jb;
                next_hits(ma, mb, &ja, &jb);
                const float4 a = sm.ta[base + ja], b = sm.ta[base + jb];
                const u64 ex = sub2(pack2(a.x, b.x), x2), ey = sub2(pack2(a.y, b.y), y2), ez = sub2(pack2(a.z, b.z), z2);
                const u64 r2 = fma2(ez, ez, fma2(ey, ey, mul2(ex, ex)));
                float r2a, r2b;
                unpack2(r2, r2a, r2b);
                // the exact cut-off; r = 0 is the particle itself.  A miss (filter false positive, dummy) is carried along
                // with r^2 = 1 and mass 0: every term stays finite and contributes exactly zero.
                const bool hitA = r2a < fmaxf(hc2A, a.w) && r2a > 0.f, hitB = r2b < fmaxf(hc2B, b.w) && r2b > 0.f;
                r2a = hitA ? r2a : 1.0f; r2b = hitB ? r2b : 1.0f;
                const u64 r2s = pack2(r2a, r2b);
                u64 rinv = pack2(rsqrtf(r2a), rsqrtf(r2b));
                rinv = mul2(rinv, fma2(mul2(mul2(kMHalf2, r2s), rinv), rinv, kOneHalf2));      // one Newton step: ~1 ulp
                const u64 r = mul2(r2s, rinv);
                const float4 va = sm.tb[base + ja], vb = sm.tb[base + jb], ca = sm.tc[base + ja], cb = sm.tc[base + jb];
                const u64 ihj = pack2(ca.w, cb.w);
                const u64 Gi = mul2(spline_dw2(mul2(r, inv_h2), kTwo, kOne, kThree, kM075), n42);
                const u64 ih2 = mul2(ihj, ihj);
                const u64 Gj = mul2(spline_dw2(mul2(r, ihj), kTwo, kOne, kThree, kM075), mul2(mul2(ih2, ih2), kInvPi2));
                const u64 wx = sub2(pack2(va.x, vb.x), vx2), wy = sub2(pack2(va.y, vb.y), vy2), wz = sub2(pack2(va.z, vb.z), vz2);
                const u64 vr = mul2(fma2(wz, ez, fma2(wy, ey, mul2(wx, ex))), rinv);
                float vra, vrb;
                unpack2(vr, vra, vrb);
                const u64 mu = pack2(fminf(vra, 0.f), fminf(vrb, 0.f));
                const u64 vs = fma2(kMBeta2, mu, add2(c2, pack2(ca.z, cb.z)));
                float rsa, rsb, vsa, vsb;
                unpack2(add2(rho2, pack2(ca.x, cb.x)), rsa, rsb);
                unpack2(vs, vsa, vsb);
                const u64 visc = mul2(mul2(mul2(kMAlpha2, vs), mu), pack2(rcp_approx(rsa), rcp_approx(rsb)));   // -(alpha/2) vs mu / ((rho_i+rho_j)/2)
                const u64 vG = mul2(mul2(visc, kHalf2), add2(Gi, Gj));
                const u64 AG = mul2(A2, Gi), BG = mul2(pack2(ca.y, cb.y), Gj);
                const u64 m = pack2(hitA ? va.w : 0.f, hitB ? vb.w : 0.f);
                const u64 fr = mul2(mul2(m, add2(add2(AG, BG), vG)), rinv);
                ax = fma2(fr, ex, ax); ay = fma2(fr, ey, ay); az = fma2(fr, ez, az);
                du = fma2(mul2(m, fma2(kHalf2, vG, AG)), vr, du);
                vsigA = fmaxf(vsigA, hitA ? vsa : 0.f); vsigB = fmaxf(vsigB, hitB ? vsb : 0.f);
            }
        };
        auto flush = [&](uint32_t cnt) {
            // filter cut-off of a target: max((2 h_i)^2, largest (2 h_j)^2 in the tile) -- a superset of max(2h_i, 2h_j) per pair
            const float cutA = fmaxf(hc2A, tile_hc2), cutB = fmaxf(hc2B, tile_hc2);
            const float b2 = 3.0f * fmaxf(tile_b2, ri2_max);
            const FilterTarget fA = filter_target(xA, yA, zA, vA ? ri2A - cutA - kFilterEps * (b2 + cutA) : kNever);
            const FilterTarget fB = filter_target(xB, yB, zB, vB ? ri2B - cutB - kFilterEps * (b2 + cutB) : kNever);
            uint32_t m[4];
            filter_masks(sm.f, cnt, lane, fA, fB, m);
            hits(m[0], m[2], 0);
            if (cnt > 32) hits(m[1], m[3], kHalf);
            tile_hc2 = 0.f; tile_b2 = 0.f;
            __syncwarp();
        };

        uint32_t cnt = 0;
        const uint32_t n_rounds = max(1u, (n_s + 31) >> 5);
        for (uint32_t r = 0; r < n_rounds; ++r) {
            const uint32_t j0 = 32 * r, nj = min(32u, n_s - j0);
            if (r > 0) { cp_async_wait_all(); __syncwarp(); }
            // one step ahead: the next round of this item (the next item's records are fetched after the results have left sm.tgt)
            if (r + 1 < n_rounds) fetch_records<13, 32>(sm.src[buf ^ 1], sin + (uint64_t)(j0 + 32) * 52, min(32u, n_s - j0 - 32), lane);
            float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a, c = a;
            float s2 = 0.f;
            bool ok = false;
            if (lane < nj) {
                const float* rec = sm.src[buf] + 13 * lane;
                const float h = rec[3], rho = rec[5];
                const float reach = fmaxf(reach_t, 2.0f * h) * kReachSlack;
                a = make_float4(rec[0], rec[1], rec[2], 4.0f * h * h);
                ok = a.x > lox - reach && a.x < hix + reach && a.y > loy - reach && a.y < hiy + reach && a.z > loz - reach && a.z < hiz + reach;
                if (ok) {
                    b = make_float4(rec[7], rec[8], rec[9], rec[4]);
                    c = make_float4(rho, rec[11] / ((1.0f + h * rec[6] / (3.0f * rho)) * rho * rho), rec[12], 1.0f / h);
                    s2 = fmaf(a.x, a.x, fmaf(a.y, a.y, a.z * a.z));
                }
            }
            const uint32_t ball = __ballot_sync(kFull, ok), n_ok = __popc(ball);
            if (cnt + n_ok > kTile) { flush(cnt); cnt = 0; }
            if (ok) {
                const uint32_t pos = cnt + __popc(ball & lt), e = pos + (pos >> 5);      // half * 33 + index in the half
                sm.ta[e] = a; sm.tb[e] = b; sm.tc[e] = c;
                filter_put(sm.f, pos, a.x, a.y, a.z, s2);
            }
            tile_hc2 = fmaxf(tile_hc2, warp_max_pos(ok ? a.w : 0.f));
            tile_b2 = fmaxf(tile_b2, warp_max_pos(s2));
            cnt += n_ok;
            buf ^= 1;
        }
        if (cnt) flush(cnt);
        // results through shared memory so the 20-byte records leave as coalesced 16-byte stores
        float axA, axB, ayA, ayB, azA, azB, duA, duB;
        unpack2(ax, axA, axB); unpack2(ay, ayA, ayB); unpack2(az, azA, azB); unpack2(du, duA, duB);
        if (vA) { float* o = sm.tgt + 5 * lane; o[0] = axA; o[1] = ayA; o[2] = azA; o[3] = duA; o[4] = vsigA; }
        if (vB) { float* o = sm.tgt + 5 * (lane + 32); o[0] = axB; o[1] = ayB; o[2] = azB; o[3] = duB; o[4] = vsigB; }
        __syncwarp();
        const uint32_t nvec = (n_t * 5 + 3) >> 2;
        for (uint32_t v = lane; v < nvec; v += 32) reinterpret_cast<uint4*>(tout)[v] = reinterpret_cast<const uint4*>(sm.tgt)[v];
        __syncwarp();
        if (has_next) {
            fetch_records<13, 64>(sm.tgt, in + (uint64_t)iw_next.x * 128, iw_next.w & 127u, lane);
            fetch_records<13, 32>(sm.src[buf], in + (uint64_t)iw_next.y * 128, min(32u, iw_next.w >> 7), lane);
        }
        iw = iw_next;
    }
}

template <class K>
int32_t loop_grid(K kernel, size_t smem, uint32_t* grid) {
    int dev = 0, sms = 0, per_sm = 0;
    SPH_CUDA_TRY(cudaGetDevice(&dev));
    SPH_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (smem > 48 * 1024) SPH_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    SPH_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kLoopWarps * 32, smem));
    *grid = (uint32_t)(sms * max(per_sm, 1));
    return SPH_OK;
}

}  // namespace

int32_t launch_density(const sph_batch* b, const char* d_in, char* d_out, cudaStream_t st) {
    if (b->n_chunks == 0) return SPH_OK;
    static uint32_t full_grid = 0;
    if (!full_grid)
        if (int32_t rc = loop_grid(density_kernel, 0, &full_grid)) return rc;
    const uint32_t grid = min((b->n_chunks + kLoopWarps - 1) / kLoopWarps, full_grid);
    density_kernel<<<grid, kLoopWarps * 32, 0, st>>>(b->d_items_density, d_in, d_out, b->n_chunks);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_force(const sph_batch* b, const char* d_in, char* d_out, const sph_params& prm, cudaStream_t st) {
    if (b->n_chunks == 0) return SPH_OK;
    static uint32_t full_grid = 0;
    constexpr size_t smem = sizeof(ForceWarpSmem) * kLoopWarps;
    if (!full_grid)
        if (int32_t rc = loop_grid(force_kernel, smem, &full_grid)) return rc;
    const uint32_t grid = min((b->n_chunks + kLoopWarps - 1) / kLoopWarps, full_grid);
    force_kernel<<<grid, kLoopWarps * 32, smem, st>>>(b->d_items_force, d_in, d_out, b->n_chunks, prm.alpha, prm.beta);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
