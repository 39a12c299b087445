// DENSITY and FORCE interaction loops over cell / cell-pair tasks.
//
// Nothing here is a dense contraction (a few percent of the candidate pairs are neighbours and the per-pair
// work is a distance test), so this is plain FP32 ALU work, not tensor-core work.
//
// Work item = (up to 64 target particles of one block, two per lane: A = lane, B = lane + 32) x (the block they
// gather from: the task's other side, or the block itself for a self task); one 16-byte item descriptor, built
// with the batch.  One warp per item, warps never wait for one another (no __syncthreads):
//   (a) records travel global -> shared memory one step AHEAD of their use -- in the force loop (52-byte records) as bulk
//       copies (TMA, cp.async.bulk: one instruction per block of records, completing on the warp's mbarrier), in the
//       density loop (20-byte records, short rounds: the start-up latency of a bulk copy is not covered there, measured
//       193 vs 181 us) as coalesced 16-byte cp.async copies:
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
//   (d) phase 2, density and gradient loops: every lane walks the set bits of its two masks in source order, one hit of
//       target A and one of target B per iteration, the pair evaluated with packed f32x2 arithmetic (a target that has
//       run out of hits is fed a far-away dummy source whose contribution is exactly zero); force loop (expensive hits,
//       heavy-tailed counts per target): the masks are cut into units of <= 4 hits evaluated 32 at a time (see the kernel).
//       r^2 = |x_i - s|^2 is recomputed exactly as the definition does and the exact cut-off applied.
// Sums are accumulated per target in tile order = source order, so results are bit-reproducible run to run.
#include "internal.h"
#include "ptx.cuh"
#include <type_traits>

namespace sph {

namespace {

using namespace ptx;           // u64 = a pair of f32 (lo = target A, hi = target B)

#ifndef SPH_LOOP_WARPS
#define SPH_LOOP_WARPS 4
#endif
#ifndef SPH_FORCE_MINB
#define SPH_FORCE_MINB 4
#endif
#ifndef SPH_DENS_MINB
#define SPH_DENS_MINB 5
#endif
#ifndef SPH_UNIT_CAP
#define SPH_UNIT_CAP 96
#endif
constexpr int kLoopWarps = SPH_LOOP_WARPS;
constexpr int kTile = 64;                  // compacted sources per flush: two halves of 32, one mask word each per target
constexpr int kHalf = 33;                  // tile entries per half: 32 sources + the dummy (where __clz(0) = 32 points)
#ifndef SPH_UNIT_BITS
#define SPH_UNIT_BITS 4
#endif
constexpr uint32_t kUnitBits = SPH_UNIT_BITS;      // neighbours per unit (even)
constexpr int kUnitCap = SPH_UNIT_CAP;               // units (target, <= 4 neighbours) evaluated per window of a flush, 32 at a time
constexpr float kInvPi = 0.318309886183790671538f;
constexpr float kNever = 1.0e30f;          // |s|^2 of a filter pad entry / threshold of an idle target: never a hit
constexpr float kFar = 1.0e15f;            // coordinates of the dummy source (r^2 = 3e30 stays finite)
constexpr float kReachSlack = 1.0f + 1.0e-4f;   // the reach box is a superset test; keep it clear of f32 rounding
constexpr float kFilterEps = 4.0e-6f;      // x (largest |coordinate|)^2 summed over the axes: bounds the rounding of the
                                           // expanded form (about 18 roundings of 2^-24 relative to that scale)
constexpr uint32_t kFull = kFullMask;

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) { cp_async<16>(smem, gmem); }

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

// bytes of n records of WORDS 4-byte words, rounded up to the 16 bytes a bulk copy moves (a last partial vector reads
// into the block's pad bytes)
template <int WORDS>
__device__ __forceinline__ uint32_t rec_bytes16(uint32_t n) { return (n * WORDS * 4 + 15) & ~15u; }

// One GROUP of record fetches, issued by lane 0 and waited for by the whole warp at the next wait point: the records are
// contiguous and 16-byte aligned in global memory, so each fetch is a single bulk copy -- no per-lane address arithmetic,
// no registers held while it is in flight.  At most one group is outstanding per warp; `parity` tracks the barrier phase.
struct FetchGroup {
    uint64_t* bar;
    uint32_t parity;
    __device__ __forceinline__ void issue1(uint32_t lane, void* d0, const void* g0, uint32_t b0) {
        fence_proxy_async();      // the destination was last read through the generic proxy
        __syncwarp();
        if (lane == 0) { mbar_expect_tx(bar, b0); if (b0) bulk_g2s(d0, g0, b0, bar); }
    }
    __device__ __forceinline__ void issue2(uint32_t lane, void* d0, const void* g0, uint32_t b0, void* d1, const void* g1, uint32_t b1) {
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) { mbar_expect_tx(bar, b0 + b1); if (b0) bulk_g2s(d0, g0, b0, bar); if (b1) bulk_g2s(d1, g1, b1, bar); }
    }
    __device__ __forceinline__ void wait() { mbar_wait(bar, parity); parity ^= 1; }
};

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

// Phase 1 over the first `cnt` tile entries for the lane's targets: bit (31 - j) of m[0] = "source j may be a
// neighbour of target A" (j < 32), m[1] likewise for sources 32..63; m[2], m[3] for target B (DUAL only).
template <bool DUAL>
__device__ __forceinline__ void filter_half(const FilterTile& f, uint32_t lo, uint32_t hi, const FilterTarget& A, const FilterTarget& B, uint32_t& ma, uint32_t& mb) {
    // the tile is padded to a multiple of eight entries (tile_box): four packed source pairs per trip, no remainder loop
#pragma unroll 1
    for (uint32_t p0 = lo; p0 < hi; p0 += 4) {
#pragma unroll
        for (uint32_t k = 0; k < 4; ++k) {
            const ulonglong2 a = *reinterpret_cast<const ulonglong2*>(&f.a[p0 + k]);
            const ulonglong2 b = *reinterpret_cast<const ulonglong2*>(&f.b[p0 + k]);
            const u64 ta = fma2(A.mx2, a.x, fma2(A.my2, a.y, fma2(A.mz2, b.x, add2(b.y, A.nt2))));
            uint32_t lo32, hi32;
            asm("mov.b64 {%0, %1}, %2;" : "=r"(lo32), "=r"(hi32) : "l"(ta));
            ma = __funnelshift_l(lo32, ma, 1);      // (m << 1) | sign(t_lo)
            ma = __funnelshift_l(hi32, ma, 1);
            if constexpr (DUAL) {
                const u64 tb = fma2(B.mx2, a.x, fma2(B.my2, a.y, fma2(B.mz2, b.x, add2(b.y, B.nt2))));
                asm("mov.b64 {%0, %1}, %2;" : "=r"(lo32), "=r"(hi32) : "l"(tb));
                mb = __funnelshift_l(lo32, mb, 1);
                mb = __funnelshift_l(hi32, mb, 1);
            }
        }
    }
}
__device__ __forceinline__ void filter_masks(const FilterTile& f, uint32_t cnt, bool dual, const FilterTarget& A, const FilterTarget& B, uint32_t (&m)[4]) {
    const uint32_t np = ((cnt + 7) & ~7u) >> 1;          // packed source pairs, a multiple of four
    // ONE copy of each loop serves both tile halves: the loops' code must stay inside the SM's instruction cache (ncu: "no
    // instruction" was the first stall reason of the r01 kernels, whose bodies were 85-115 KB)
#pragma unroll 1
    for (uint32_t h = 0; h < 2; ++h) {
        const uint32_t lo = 16 * h, hi = min(np, lo + 16);
        uint32_t ma = 0, mb = 0;
        if (hi > lo) {
            if (dual) filter_half<true>(f, lo, hi, A, B, ma, mb); else filter_half<false>(f, lo, hi, A, B, ma, mb);
            ma <<= 32 - 2 * (hi - lo); mb <<= 32 - 2 * (hi - lo);
        }
        if (h == 0) { m[0] = ma; m[2] = mb; } else { m[1] = ma; m[3] = mb; }
    }
}

// pads the filter tile to a multiple of eight entries and returns the bounding box of its first cnt sources
struct Box { float lox, hix, loy, hiy, loz, hiz; };
__device__ __forceinline__ Box tile_box(FilterTile& f, uint32_t cnt, uint32_t lane) {
    const uint32_t n8 = (cnt + 7) & ~7u;
    if (lane < n8 - cnt) filter_put(f, cnt + lane, 0.f, 0.f, 0.f, kNever);
    __syncwarp();
    // entries lane and lane + 32 of the tile
    const float* a = reinterpret_cast<const float*>(&f.a[lane >> 1]) + (lane & 1);
    const float* b = reinterpret_cast<const float*>(&f.b[lane >> 1]) + (lane & 1);
    const bool v0 = lane < cnt, v1 = lane + 32 < cnt;
    const float x0 = a[0], y0 = a[2], z0 = b[0];
    const float x1 = v1 ? a[64] : x0, y1 = v1 ? a[66] : y0, z1 = v1 ? b[64] : z0;      // + 16 float4 = + 64 floats
    Box bx;
    bx.lox = warp_min(fminf(x0, x1), v0); bx.hix = warp_max(fmaxf(x0, x1), v0);
    bx.loy = warp_min(fminf(y0, y1), v0); bx.hiy = warp_max(fmaxf(y0, y1), v0);
    bx.loz = warp_min(fminf(z0, z1), v0); bx.hiz = warp_max(fmaxf(z0, z1), v0);
    return bx;
}
// squared distance from a point to a box
__device__ __forceinline__ float box_dist2(const Box& b, float x, float y, float z) {
    const float dx = fmaxf(fmaxf(b.lox - x, x - b.hix), 0.f), dy = fmaxf(fmaxf(b.loy - y, y - b.hiy), 0.f), dz = fmaxf(fmaxf(b.loz - z, z - b.hiz), 0.f);
    return fmaf(dz, dz, fmaf(dy, dy, dx * dx));
}

// the next two hits of a pass: of targets A and B (dual), or the next two of target A (single); 32 = the dummy
__device__ __forceinline__ bool next_hits(bool dual, uint32_t& ma, uint32_t& mb, uint32_t* ja, uint32_t* jb) {
    if (dual) {
        if ((ma | mb) == 0) return false;
        *ja = __clz(ma); *jb = __clz(mb);
        ma &= ~shr_clamp(0x80000000u, *ja);
        mb &= ~shr_clamp(0x80000000u, *jb);
    } else {
        if (ma == 0) return false;
        *ja = __clz(ma);
        ma &= ~shr_clamp(0x80000000u, *ja);
        *jb = __clz(ma);
        ma &= ~shr_clamp(0x80000000u, *jb);
    }
    return true;
}

// Which of the item's targets can have a neighbour in the tile: the active ones are numbered through (A targets
// first, lane order) into sm_act; returns their count.  aA / aB: is the lane's own target lane / lane + 32 active.
__device__ __forceinline__ uint32_t compact_targets(uint32_t* sm_act, bool aA, bool aB, uint32_t lane, uint32_t lt) {
    const uint32_t bA = __ballot_sync(kFull, aA), bB = __ballot_sync(kFull, aB), nA = __popc(bA);
    if (aA) sm_act[__popc(bA & lt)] = lane;
    if (aB) sm_act[nA + __popc(bB & lt)] = lane + 32;
    __syncwarp();
    return nA + __popc(bB);
}

// Cell-slot records: x travels as raw f64 (words 0-5) and the frame of the item's side is applied here,
// exactly as the pack applies it -- one f64 subtraction, one rounding -- so a loop over slots sees bit for bit the inputs of
// a loop over per-task records.  Every other field sits three words further on; a last word (time_bin) makes the record
// length odd (9 / 17 words), so that one record per lane reads conflict-free out of the landing area.
template <bool SLOTS>
__device__ __forceinline__ float rec_x(const float* r, int d, const double* frame) {
    if constexpr (SLOTS) return (float)(__hiloint2double(__float_as_int(r[2 * d + 1]), __float_as_int(r[2 * d])) - frame[d]);
    else return r[d];
}

// ------------------------------------------------------------------------------------------------- density

template <int RW>
struct DensityWarpSmemT {
    FilterTile f;
    float4 tile[2 * kHalf];  // x, y, z, m of the compacted sources; entries 32 and 65 are the dummy
    float4 tgt[64];          // the item's targets: x, y, z, h
    float4 acc[64];          // their running sums: m w, m (3w + q w'), w, (3w + q w')
    float raw[64 * RW];      // landing area of an item's 64 DENSITY_IN records: xr0 xr1 xr2 h m (slots: x f64[3] h m time_bin)
    float src[2][32 * RW];   // landing areas of the source rounds (double-buffered)
    uint32_t act[64];        // the active targets of the flush
};

template <bool SLOTS>
__global__ void __launch_bounds__(kLoopWarps * 32, SPH_DENS_MINB)
density_kernel(const LoopItem* __restrict__ items, const char* __restrict__ in, char* __restrict__ out, uint32_t n_items,
               const double* __restrict__ item_frames) {
    constexpr int RW = SLOTS ? 9 : 5, O = SLOTS ? 3 : 0;      // record words; offset of the fields behind x
    typedef DensityWarpSmemT<RW> DensityWarpSmem;
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
    fetch_records<RW, 64>(sm.raw, in + (uint64_t)iw.x * 128, iw.w & 127u, lane);
    fetch_records<RW, 32>(sm.src[0], in + (uint64_t)iw.y * 128, min(32u, iw.w >> 7), lane);
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
        // the lane's own two targets (lane, lane + 32): table entries, zeroed sums, reach box of the whole item
        const bool vA = lane < n_t, vB = lane + 32 < n_t;
        double ft[3] = {0.0, 0.0, 0.0}, fs[3] = {0.0, 0.0, 0.0};      // slots: the frames of the targets' and of the sources' side
        if constexpr (SLOTS) {
#pragma unroll
            for (int d = 0; d < 3; ++d) { ft[d] = __ldg(item_frames + 6 * (size_t)item + d); fs[d] = __ldg(item_frames + 6 * (size_t)item + 3 + d); }
        }
        float4 oA = make_float4(0.f, 0.f, 0.f, 0.f), oB = oA;
        if (vA) { const float* r = sm.raw + RW * lane; oA = make_float4(rec_x<SLOTS>(r, 0, ft), rec_x<SLOTS>(r, 1, ft), rec_x<SLOTS>(r, 2, ft), r[3 + O]); }
        if (vB) { const float* r = sm.raw + RW * (lane + 32); oB = make_float4(rec_x<SLOTS>(r, 0, ft), rec_x<SLOTS>(r, 1, ft), rec_x<SLOTS>(r, 2, ft), r[3 + O]); }
        sm.tgt[lane] = oA; sm.tgt[lane + 32] = oB;
        sm.acc[lane] = make_float4(0.f, 0.f, 0.f, 0.f); sm.acc[lane + 32] = make_float4(0.f, 0.f, 0.f, 0.f);
        __syncwarp();                 // sm.raw may now receive the next item's targets
        const float reach = 2.0f * warp_max_pos(fmaxf(oA.w, oB.w)) * kReachSlack;
        const float lox = warp_min(vB ? fminf(oA.x, oB.x) : oA.x, vA) - reach, hix = warp_max(vB ? fmaxf(oA.x, oB.x) : oA.x, vA) + reach;
        const float loy = warp_min(vB ? fminf(oA.y, oB.y) : oA.y, vA) - reach, hiy = warp_max(vB ? fmaxf(oA.y, oB.y) : oA.y, vA) + reach;
        const float loz = warp_min(vB ? fminf(oA.z, oB.z) : oA.z, vA) - reach, hiz = warp_max(vB ? fmaxf(oA.z, oB.z) : oA.z, vA) + reach;
        const float bx = fmaxf(fabsf(lox), fabsf(hix)), by = fmaxf(fabsf(loy), fabsf(hiy)), bz = fmaxf(fabsf(loz), fabsf(hiz));
        const float eps = kFilterEps * fmaf(bx, bx, fmaf(by, by, bz * bz));
        const float cutA = 4.0f * oA.w * oA.w, cutB = 4.0f * oB.w * oB.w;

        auto flush = [&](uint32_t cnt) {
            // targets that can reach the tile's bounding box get a lane (or half of one); the others sit this flush out
            const Box box = tile_box(sm.f, cnt, lane);
            const bool aA = vA && box_dist2(box, oA.x, oA.y, oA.z) < cutA * kReachSlack, aB = vB && box_dist2(box, oB.x, oB.y, oB.z) < cutB * kReachSlack;
            const uint32_t n_act = compact_targets(sm.act, aA, aB, lane, lt);
            if (n_act == 0) return;
            const bool dual = n_act > 32;                // else: one target per lane, two of its hits per iteration
            const bool wA = lane < n_act, wB = dual && lane + 32 < n_act;
            const uint32_t tA = wA ? sm.act[lane] : 0, tB = wB ? sm.act[lane + 32] : tA;
            const float4 pA = sm.tgt[tA], pB = sm.tgt[tB];
            const float inv_hA = wA ? rcp_fast(pA.w) : 0.f, inv_hB = dual ? (wB ? rcp_fast(pB.w) : 0.f) : inv_hA;
            const FilterTarget fA = filter_target(pA.x, pA.y, pA.z, wA ? fmaf(pA.x, pA.x, fmaf(pA.y, pA.y, pA.z * pA.z)) - 4.0f * pA.w * pA.w - eps : kNever);
            const FilterTarget fB = filter_target(pB.x, pB.y, pB.z, wB ? fmaf(pB.x, pB.x, fmaf(pB.y, pB.y, pB.z * pB.z)) - 4.0f * pB.w * pB.w - eps : kNever);
            uint32_t m[4];
            filter_masks(sm.f, cnt, dual, fA, fB, m);
            const u64 x2 = pack2(pA.x, pB.x), y2 = pack2(pA.y, pB.y), z2 = pack2(pA.z, pB.z);
            u64 s_mw = 0, s_mg = 0, s_w = 0, s_g = 0;
            // phase 2 over one half of the tile
            auto hits = [&](uint32_t ma, uint32_t mb, const float4* half) {
                uint32_t ja, jb;
                while (next_hits(dual, ma, mb, &ja, &jb)) {
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
                    const u64 mm = pack2(a.w, b.w);
                    s_mw = fma2(mm, w, s_mw); s_mg = fma2(mm, g, s_mg);
                    s_w = add2(s_w, w); s_g = add2(s_g, g);
                }
            };
#pragma unroll 1
            for (uint32_t h = 0; h < 2 && 32 * h < cnt; ++h) hits(h ? m[1] : m[0], h ? m[3] : m[2], sm.tile + h * kHalf);
            float mw0, mw1, mg0, mg1, w0, w1, g0, g1;
            unpack2(s_mw, mw0, mw1); unpack2(s_mg, mg0, mg1); unpack2(s_w, w0, w1); unpack2(s_g, g0, g1);
            if (dual) {
                if (wA) { float4 c = sm.acc[tA]; c.x += mw0; c.y += mg0; c.z += w0; c.w += g0; sm.acc[tA] = c; }
                if (wB) { float4 c = sm.acc[tB]; c.x += mw1; c.y += mg1; c.z += w1; c.w += g1; sm.acc[tB] = c; }
            } else if (wA) {
                float4 c = sm.acc[tA];
                c.x += mw0 + mw1; c.y += mg0 + mg1; c.z += w0 + w1; c.w += g0 + g1;
                sm.acc[tA] = c;
            }
        };

        uint32_t cnt = 0;
        const uint32_t n_rounds = max(1u, (n_s + 31) >> 5);
        // round n_rounds is the closing one: nothing new, what is left in the tile is flushed (one flush site: code size)
        for (uint32_t r = 0; r <= n_rounds; ++r) {
            float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
            bool ok = false;
            uint32_t ball = 0, c = 0;
            if (r < n_rounds) {
                const uint32_t j0 = 32 * r, nj = min(32u, n_s - j0);
                if (r > 0) { cp_async_wait_all(); __syncwarp(); }
                // one step ahead: the next round of this item, or the next item's targets and first round
                if (r + 1 < n_rounds) {
                    fetch_records<RW, 32>(sm.src[buf ^ 1], sin + (uint64_t)(j0 + 32) * (RW * 4), min(32u, n_s - j0 - 32), lane);
                } else if (has_next) {
                    fetch_records<RW, 64>(sm.raw, in + (uint64_t)iw_next.x * 128, iw_next.w & 127u, lane);
                    fetch_records<RW, 32>(sm.src[buf ^ 1], in + (uint64_t)iw_next.y * 128, min(32u, iw_next.w >> 7), lane);
                }
                if (lane < nj) {
                    const float* rec = sm.src[buf] + RW * lane;
                    s = make_float4(rec_x<SLOTS>(rec, 0, fs), rec_x<SLOTS>(rec, 1, fs), rec_x<SLOTS>(rec, 2, fs), rec[4 + O]);
                    ok = s.x > lox && s.x < hix && s.y > loy && s.y < hiy && s.z > loz && s.z < hiz;
                }
                ball = __ballot_sync(kFull, ok); c = __popc(ball);
            }
            if (cnt + c > kTile || (r == n_rounds && cnt)) { flush(cnt); __syncwarp(); cnt = 0; }
            if (ok) {
                const uint32_t pos = cnt + __popc(ball & lt);
                sm.tile[pos + (pos >> 5)] = s;        // half * 33 + index in the half
                filter_put(sm.f, pos, s.x, s.y, s.z, fmaf(s.x, s.x, fmaf(s.y, s.y, s.z * s.z)));
            }
            cnt += c;
            buf ^= r < n_rounds;
        }
        __syncwarp();
        if (vA) {
            const float ih = rcp_fast(oA.w), n3 = kInvPi * ih * ih * ih, n4 = n3 * ih;
            const float4 c = sm.acc[lane];
            reinterpret_cast<float4*>(tout)[lane] = make_float4(c.x * n3, -c.y * n4, c.z * n3, -c.w * n4);
        }
        if (vB) {
            const float ih = rcp_fast(oB.w), n3 = kInvPi * ih * ih * ih, n4 = n3 * ih;
            const float4 c = sm.acc[lane + 32];
            reinterpret_cast<float4*>(tout)[lane + 32] = make_float4(c.x * n3, -c.y * n4, c.z * n3, -c.w * n4);
        }
        __syncwarp();                 // sm.tgt / sm.acc are rewritten by the next item
        iw = iw_next;
    }
}

// ------------------------------------------------------------------------------------------------- gradient
//
// The third loop of the Sphenix-like cycle (reading C34): velocity divergence and curl with the
// volume-weighted estimators, for instance i over j != i with r < 2 h_i:
//   g = (m_j / rho_j) dW/dr(r, h_i),  e = (x_i - x_j) / r,  dv = v_j - v_i,  div_v += g (dv . e),  rot_v += g (e x dv).
// Same shape as the density loop (one-sided cut-off 2 h_i, four sums per target), another hit body and wider records:
// GRADIENT_IN = [xr0 xr1 xr2 v0 v1 v2 mass h u rho] (40 bytes), GRADIENT_OUT = [div_v rot_v0 rot_v1 rot_v2] (16 bytes).
struct GradientWarpSmem {
    FilterTile f;
    float4 tile[2 * kHalf];  // x, y, z, m / rho of the compacted sources; entries 32 and 65 are the dummy
    float4 tilev[2 * kHalf]; // their vx, vy, vz
    float4 tgt[64];          // the item's targets: x, y, z, h
    float4 tgv[64];          //                     vx, vy, vz
    float4 acc[64];          // their running sums: div, rot (3), before the 1 / (pi h^4)
    float raw[64 * 10];      // landing area of an item's 64 GRADIENT_IN records
    float src[2][32 * 10];   // landing areas of the source rounds (double-buffered)
    uint32_t act[64];        // the active targets of the flush
};

__global__ void __launch_bounds__(kLoopWarps * 32, 3)
gradient_kernel(const LoopItem* __restrict__ items, const char* __restrict__ in, char* __restrict__ out, uint32_t n_items) {
    extern __shared__ __align__(16) unsigned char s_raw[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    GradientWarpSmem& sm = reinterpret_cast<GradientWarpSmem*>(s_raw)[warp];
    const uint32_t lt = lanemask_lt();
    const uint32_t step = gridDim.x * kLoopWarps;
    uint32_t item = blockIdx.x * kLoopWarps + warp;
    if (item >= n_items) return;
    if (lane < 2) { sm.tile[lane * kHalf + 32] = make_float4(kFar, kFar, kFar, 0.f); sm.tilev[lane * kHalf + 32] = make_float4(0.f, 0.f, 0.f, 0.f); }
    const u64 kTwo = dup2(2.0f), kOne = dup2(1.0f), kThree = dup2(3.0f), kM075 = dup2(-0.75f);

    uint4 iw = __ldg(reinterpret_cast<const uint4*>(items) + item);
    fetch_records<10, 64>(sm.raw, in + (uint64_t)iw.x * 128, iw.w & 127u, lane);
    fetch_records<10, 32>(sm.src[0], in + (uint64_t)iw.y * 128, min(32u, iw.w >> 7), lane);
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
        float4 oA = make_float4(0.f, 0.f, 0.f, 0.f), oB = oA, wA4 = oA, wB4 = oA;
        if (vA) { const float* r = sm.raw + 10 * lane; oA = make_float4(r[0], r[1], r[2], r[7]); wA4 = make_float4(r[3], r[4], r[5], 0.f); }
        if (vB) { const float* r = sm.raw + 10 * (lane + 32); oB = make_float4(r[0], r[1], r[2], r[7]); wB4 = make_float4(r[3], r[4], r[5], 0.f); }
        sm.tgt[lane] = oA; sm.tgt[lane + 32] = oB; sm.tgv[lane] = wA4; sm.tgv[lane + 32] = wB4;
        sm.acc[lane] = make_float4(0.f, 0.f, 0.f, 0.f); sm.acc[lane + 32] = make_float4(0.f, 0.f, 0.f, 0.f);
        __syncwarp();                 // sm.raw may now receive the next item's targets
        const float reach = 2.0f * warp_max_pos(fmaxf(oA.w, oB.w)) * kReachSlack;
        const float lox = warp_min(vB ? fminf(oA.x, oB.x) : oA.x, vA) - reach, hix = warp_max(vB ? fmaxf(oA.x, oB.x) : oA.x, vA) + reach;
        const float loy = warp_min(vB ? fminf(oA.y, oB.y) : oA.y, vA) - reach, hiy = warp_max(vB ? fmaxf(oA.y, oB.y) : oA.y, vA) + reach;
        const float loz = warp_min(vB ? fminf(oA.z, oB.z) : oA.z, vA) - reach, hiz = warp_max(vB ? fmaxf(oA.z, oB.z) : oA.z, vA) + reach;
        const float bx = fmaxf(fabsf(lox), fabsf(hix)), by = fmaxf(fabsf(loy), fabsf(hiy)), bz = fmaxf(fabsf(loz), fabsf(hiz));
        const float eps = kFilterEps * fmaf(bx, bx, fmaf(by, by, bz * bz));
        const float cutA = 4.0f * oA.w * oA.w, cutB = 4.0f * oB.w * oB.w;

        auto flush = [&](uint32_t cnt) {
            const Box box = tile_box(sm.f, cnt, lane);
            const bool aA = vA && box_dist2(box, oA.x, oA.y, oA.z) < cutA * kReachSlack, aB = vB && box_dist2(box, oB.x, oB.y, oB.z) < cutB * kReachSlack;
            const uint32_t n_act = compact_targets(sm.act, aA, aB, lane, lt);
            if (n_act == 0) return;
            const bool dual = n_act > 32;
            const bool wA = lane < n_act, wB = dual && lane + 32 < n_act;
            const uint32_t tA = wA ? sm.act[lane] : 0, tB = wB ? sm.act[lane + 32] : tA;
            const float4 pA = sm.tgt[tA], pB = sm.tgt[tB], qA = sm.tgv[tA], qB = sm.tgv[tB];
            const float inv_hA = wA ? rcp_fast(pA.w) : 0.f, inv_hB = dual ? (wB ? rcp_fast(pB.w) : 0.f) : inv_hA;
            const FilterTarget fA = filter_target(pA.x, pA.y, pA.z, wA ? fmaf(pA.x, pA.x, fmaf(pA.y, pA.y, pA.z * pA.z)) - 4.0f * pA.w * pA.w - eps : kNever);
            const FilterTarget fB = filter_target(pB.x, pB.y, pB.z, wB ? fmaf(pB.x, pB.x, fmaf(pB.y, pB.y, pB.z * pB.z)) - 4.0f * pB.w * pB.w - eps : kNever);
            uint32_t m[4];
            filter_masks(sm.f, cnt, dual, fA, fB, m);
            const u64 x2 = pack2(pA.x, pB.x), y2 = pack2(pA.y, pB.y), z2 = pack2(pA.z, pB.z);
            const u64 vx2 = pack2(qA.x, qB.x), vy2 = pack2(qA.y, qB.y), vz2 = pack2(qA.z, qB.z), ih2 = pack2(inv_hA, inv_hB);
            u64 s_d = 0, s_x = 0, s_y = 0, s_z = 0;
            auto hits = [&](uint32_t ma, uint32_t mb, uint32_t base) {
                uint32_t ja, jb;
                while (next_hits(dual, ma, mb, &ja, &jb)) {
                    const float4 a = sm.tile[base + ja], b = sm.tile[base + jb], va = sm.tilev[base + ja], vb = sm.tilev[base + jb];
                    // d = x_i - x_j; e = d / r; dv = v_j - v_i
                    const u64 dx = sub2(x2, pack2(a.x, b.x)), dy = sub2(y2, pack2(a.y, b.y)), dz = sub2(z2, pack2(a.z, b.z));
                    const u64 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
                    float r2a, r2b;
                    unpack2(r2, r2a, r2b);
                    // r = 0 is the particle itself (d = 0: every term vanishes); the floor keeps 1 / r finite
                    const u64 rinv = pack2(rsqrtf(fmaxf(r2a, 1.0e-30f)), rsqrtf(fmaxf(r2b, 1.0e-30f)));
                    const u64 r = mul2(r2, rinv);
                    // q >= 2 (a filter false positive, the dummy): w' = 0 exactly
                    float qa, qb;
                    unpack2(mul2(r, ih2), qa, qb);
                    const u64 q = pack2(fminf(qa, 2.0f), fminf(qb, 2.0f));
                    float ta, tb, ua, ub;
                    unpack2(sub2(kTwo, q), ta, tb);
                    unpack2(sub2(kOne, q), ua, ub);
                    const u64 t = pack2(ta, tb), u = pack2(fmaxf(ua, 0.f), fmaxf(ub, 0.f));
                    const u64 dw = fma2(kThree, mul2(u, u), mul2(kM075, mul2(t, t)));      // -0.75 (2 - q)^2 + 3 (1 - q)+^2
                    const u64 g = mul2(mul2(pack2(a.w, b.w), dw), rinv);                    // (m_j / rho_j) w'(q) / r: e = d / r folded in
                    const u64 wx = sub2(pack2(va.x, vb.x), vx2), wy = sub2(pack2(va.y, vb.y), vy2), wz = sub2(pack2(va.z, vb.z), vz2);
                    s_d = fma2(g, fma2(wz, dz, fma2(wy, dy, mul2(wx, dx))), s_d);
                    s_x = fma2(g, sub2(mul2(dy, wz), mul2(dz, wy)), s_x);
                    s_y = fma2(g, sub2(mul2(dz, wx), mul2(dx, wz)), s_y);
                    s_z = fma2(g, sub2(mul2(dx, wy), mul2(dy, wx)), s_z);
                }
            };
#pragma unroll 1
            for (uint32_t h = 0; h < 2 && 32 * h < cnt; ++h) hits(h ? m[1] : m[0], h ? m[3] : m[2], h * kHalf);
            float d0, d1, x0, x1, y0, y1, z0, z1;
            unpack2(s_d, d0, d1); unpack2(s_x, x0, x1); unpack2(s_y, y0, y1); unpack2(s_z, z0, z1);
            if (dual) {
                if (wA) { float4 c = sm.acc[tA]; c.x += d0; c.y += x0; c.z += y0; c.w += z0; sm.acc[tA] = c; }
                if (wB) { float4 c = sm.acc[tB]; c.x += d1; c.y += x1; c.z += y1; c.w += z1; sm.acc[tB] = c; }
            } else if (wA) {
                float4 c = sm.acc[tA];
                c.x += d0 + d1; c.y += x0 + x1; c.z += y0 + y1; c.w += z0 + z1;
                sm.acc[tA] = c;
            }
        };

        uint32_t cnt = 0;
        const uint32_t n_rounds = max(1u, (n_s + 31) >> 5);
        for (uint32_t r = 0; r <= n_rounds; ++r) {      // round n_rounds: the closing flush (one flush site)
            float4 s = make_float4(0.f, 0.f, 0.f, 0.f), sv = s;
            bool ok = false;
            uint32_t ball = 0, c = 0;
            if (r < n_rounds) {
                const uint32_t j0 = 32 * r, nj = min(32u, n_s - j0);
                if (r > 0) { cp_async_wait_all(); __syncwarp(); }
                if (r + 1 < n_rounds) {
                    fetch_records<10, 32>(sm.src[buf ^ 1], sin + (uint64_t)(j0 + 32) * 40, min(32u, n_s - j0 - 32), lane);
                } else if (has_next) {
                    fetch_records<10, 64>(sm.raw, in + (uint64_t)iw_next.x * 128, iw_next.w & 127u, lane);
                    fetch_records<10, 32>(sm.src[buf ^ 1], in + (uint64_t)iw_next.y * 128, min(32u, iw_next.w >> 7), lane);
                }
                if (lane < nj) {
                    const float* rec = sm.src[buf] + 10 * lane;
                    s = make_float4(rec[0], rec[1], rec[2], 0.f);
                    ok = s.x > lox && s.x < hix && s.y > loy && s.y < hiy && s.z > loz && s.z < hiz;
                    if (ok) { s.w = rec[6] * rcp_fast(rec[9]); sv = make_float4(rec[3], rec[4], rec[5], 0.f); }
                }
                ball = __ballot_sync(kFull, ok); c = __popc(ball);
            }
            if (cnt + c > kTile || (r == n_rounds && cnt)) { flush(cnt); __syncwarp(); cnt = 0; }
            if (ok) {
                const uint32_t pos = cnt + __popc(ball & lt), e = pos + (pos >> 5);
                sm.tile[e] = s; sm.tilev[e] = sv;
                filter_put(sm.f, pos, s.x, s.y, s.z, fmaf(s.x, s.x, fmaf(s.y, s.y, s.z * s.z)));
            }
            cnt += c;
            buf ^= r < n_rounds;
        }
        __syncwarp();
        if (vA) {
            const float ih = rcp_fast(oA.w), n4 = kInvPi * (ih * ih) * (ih * ih);
            const float4 c = sm.acc[lane];
            reinterpret_cast<float4*>(tout)[lane] = make_float4(c.x * n4, c.y * n4, c.z * n4, c.w * n4);
        }
        if (vB) {
            const float ih = rcp_fast(oB.w), n4 = kInvPi * (ih * ih) * (ih * ih);
            const float4 c = sm.acc[lane + 32];
            reinterpret_cast<float4*>(tout)[lane + 32] = make_float4(c.x * n4, c.y * n4, c.z * n4, c.w * n4);
        }
        __syncwarp();
        iw = iw_next;
    }
}

// ------------------------------------------------------------------------------------------------- force

struct NoSwitchSmem {};
struct SwitchSmem {
    float tB[64];            // targets: Balsara factor (three-loop cycle only)
    float sB[2 * kHalf];     // sources: the same
};
template <int RW>
struct ForceWarpSmemT : std::conditional<RW == 18, SwitchSmem, NoSwitchSmem>::type {
    FilterTile f;
    float4 ta[2 * kHalf];    // sources: x, y, z, 4 h^2           (entries 32 and 65: the dummy)
    float4 tb[2 * kHalf];    //          vx, vy, vz, m
    float4 tc[2 * kHalf];    //          rho, A = P / (Omega rho^2), c_s, 1/h
    float4 t0[64];           // targets: x, y, z, 4 h^2
    float4 t1[64];           //          vx, vy, vz, c_s
    float4 t2[64];           //          1/h, 1/(pi h^4), rho, A
    float raw[64 * RW];      // landing area of an item's 64 FORCE_IN records: xr0 xr1 xr2 h m rho rho_dh v0 v1 v2 u P cs;
                             // once the target table is built: the 64 x 5 running results, in FORCE_OUT record layout
    float src[2][32 * RW];   // landing areas of the source rounds (double-buffered)
    uint32_t act[64];        // the active targets of the flush
    uint64_t bar[2];         // [0]: the mbarrier the record fetches complete on
};
typedef ForceWarpSmemT<13> ForceWarpSmem;

// -0.75 (2 - q)+^2 + 3 (1 - q)+^2 = w'(q) of the cubic spline for a pair of q
__device__ __forceinline__ u64 spline_dw2(u64 q, u64 kTwo, u64 kOne, u64 kThree, u64 kM075) {
    float ta, tb, ua, ub;
    unpack2(sub2(kTwo, q), ta, tb);
    unpack2(sub2(kOne, q), ua, ub);
    const u64 t = pack2(fmaxf(ta, 0.f), fmaxf(tb, 0.f)), u = pack2(fmaxf(ua, 0.f), fmaxf(ub, 0.f));
    return fma2(kThree, mul2(u, u), mul2(kM075, mul2(t, t)));
}

// The force terms of two (target, neighbour) pairs in packed f32x2 arithmetic (lo: first pair, hi: second pair).
// e = x_j - x_i and v_j - v_i are used (both signs flipped): (v_i - v_j).(x_i - x_j) is the same number and
// a_i += -m (..) (x_i - x_j) / r becomes one fma with e:  a_i += fr * e,  du_i += dg * vr,  v_sig_i = max(v_sig_i, vs).
struct ForceTargets2 {      // the targets' constants, one target per half
    u64 x, y, z, vx, vy, vz, cs, inv_h, n4, rho, A;
    float hc2a, hc2b;       // (2 h_i)^2
    u64 B;                  // Balsara factors (three-loop cycle; unused otherwise)
};
struct ForcePair2 {
    u64 fr, ex, ey, ez, dg, vr;
    float vsa, vsb;         // the pair's signal velocity, 0 for a miss
};
struct ForceConsts2 {
    u64 two, one, three, m075, half, mhalf, onehalf, invpi, mbeta, malpha;
};
template <bool SWITCH = false>
__device__ __forceinline__ ForcePair2 force_pair2(const ForceTargets2& T, const ForceConsts2& K, const float4& a, const float4& b,
                                                  const float4& va, const float4& vb, const float4& ca, const float4& cb, u64 Bj = 0) {
    ForcePair2 o;
    o.ex = sub2(pack2(a.x, b.x), T.x); o.ey = sub2(pack2(a.y, b.y), T.y); o.ez = sub2(pack2(a.z, b.z), T.z);
    const u64 r2 = fma2(o.ez, o.ez, fma2(o.ey, o.ey, mul2(o.ex, o.ex)));
    float r2a, r2b;
    unpack2(r2, r2a, r2b);
    // the exact cut-off; r = 0 is the particle itself.  A miss (filter false positive, dummy) is carried along
    // with r^2 = 1 and mass 0: every term stays finite and contributes exactly zero.
    const bool hitA = r2a < fmaxf(T.hc2a, a.w) && r2a > 0.f, hitB = r2b < fmaxf(T.hc2b, b.w) && r2b > 0.f;
    r2a = hitA ? r2a : 1.0f; r2b = hitB ? r2b : 1.0f;
    const u64 r2s = pack2(r2a, r2b);
    u64 rinv = pack2(rsqrtf(r2a), rsqrtf(r2b));
    rinv = mul2(rinv, fma2(mul2(mul2(K.mhalf, r2s), rinv), rinv, K.onehalf));      // one Newton step: ~1 ulp
    const u64 r = mul2(r2s, rinv);
    const u64 ihj = pack2(ca.w, cb.w);
    const u64 Gi = mul2(spline_dw2(mul2(r, T.inv_h), K.two, K.one, K.three, K.m075), T.n4);
    const u64 ih2 = mul2(ihj, ihj);
    const u64 Gj = mul2(spline_dw2(mul2(r, ihj), K.two, K.one, K.three, K.m075), mul2(mul2(ih2, ih2), K.invpi));
    const u64 wx = sub2(pack2(va.x, vb.x), T.vx), wy = sub2(pack2(va.y, vb.y), T.vy), wz = sub2(pack2(va.z, vb.z), T.vz);
    o.vr = mul2(fma2(wz, o.ez, fma2(wy, o.ey, mul2(wx, o.ex))), rinv);
    float vra, vrb;
    unpack2(o.vr, vra, vrb);
    const u64 mu = pack2(fminf(vra, 0.f), fminf(vrb, 0.f));
    const u64 vs = fma2(K.mbeta, mu, add2(T.cs, pack2(ca.z, cb.z)));
    float rsa, rsb, vsa, vsb;
    unpack2(add2(T.rho, pack2(ca.x, cb.x)), rsa, rsb);
    unpack2(vs, vsa, vsb);
    u64 visc = mul2(mul2(mul2(K.malpha, vs), mu), pack2(rcp_approx(rsa), rcp_approx(rsb)));   // -(alpha/2) vs mu / ((rho_i+rho_j)/2)
    if constexpr (SWITCH) visc = mul2(visc, mul2(K.half, add2(T.B, Bj)));                            // Balsara: (B_i + B_j) / 2
    const u64 vG = mul2(mul2(visc, K.half), add2(Gi, Gj));
    const u64 AG = mul2(T.A, Gi), BG = mul2(pack2(ca.y, cb.y), Gj);
    const u64 mm = pack2(hitA ? va.w : 0.f, hitB ? vb.w : 0.f);
    o.fr = mul2(mul2(mm, add2(add2(AG, BG), vG)), rinv);
    o.dg = mul2(mm, fma2(K.half, vG, AG));
    o.vsa = hitA ? vsa : 0.f; o.vsb = hitB ? vsb : 0.f;
    return o;
}

// Balsara-type switch (reading C34): B = |div v| / (|div v| + |rot v| + 1e-4 c_s / h)
__device__ __forceinline__ float balsara(const float* r) {      // r: a FORCE3_IN record
    const float div = fabsf(r[13]), rot = sqrtf(fmaf(r[14], r[14], fmaf(r[15], r[15], r[16] * r[16])));
    return div * rcp_fast(div + rot + 1.0e-4f * r[12] * rcp_fast(r[3]));
}

// the Balsara factors of two targets (tgt) or two tile entries, packed; nothing without the switch
template <bool SWITCH, class Smem>
__device__ __forceinline__ u64 switch_pair(const Smem& sm, uint32_t a, uint32_t b, bool tgt) {
    if constexpr (SWITCH) return tgt ? pack2(sm.tB[a], sm.tB[b]) : pack2(sm.sB[a], sm.sB[b]);
    else return 0ull;
}

template <bool SWITCH, bool SLOTS>
__global__ void __launch_bounds__(kLoopWarps * 32, SPH_FORCE_MINB)
force_kernel(const LoopItem* __restrict__ items, const char* __restrict__ in, char* __restrict__ out, uint32_t n_items, float alpha, float beta,
             const double* __restrict__ item_frames) {
    extern __shared__ __align__(16) unsigned char s_raw[];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    static_assert(!(SWITCH && SLOTS), "the switched force loop has no slot variant");
    constexpr int RW = SLOTS ? 17 : (SWITCH ? 18 : 13);      // words of an input record: FORCE_IN, FORCE3_IN = FORCE_IN + div_v rot_v[3] time_bin, or a cell slot
    constexpr int O = SLOTS ? 3 : 0;                          // slots: x is f64[3], every other field three words further on
    typedef ForceWarpSmemT<RW> Smem;
    Smem& sm = reinterpret_cast<Smem*>(s_raw)[warp];
    const uint32_t lt = lanemask_lt();
    const uint32_t step = gridDim.x * kLoopWarps;
    uint32_t item = blockIdx.x * kLoopWarps + warp;
    if (item >= n_items) return;
    if (lane < 2) {
        sm.ta[lane * kHalf + 32] = make_float4(kFar, kFar, kFar, 0.f);
        sm.tb[lane * kHalf + 32] = make_float4(0.f, 0.f, 0.f, 0.f);
        sm.tc[lane * kHalf + 32] = make_float4(0.f, 0.f, 0.f, 0.f);
        if constexpr (SWITCH) sm.sB[lane * kHalf + 32] = 0.f;
    }
    const ForceConsts2 K{dup2(2.0f), dup2(1.0f), dup2(3.0f), dup2(-0.75f), dup2(0.5f), dup2(-0.5f), dup2(1.5f), dup2(kInvPi), dup2(-beta), dup2(-alpha)};

    uint4 iw = __ldg(reinterpret_cast<const uint4*>(items) + item);
    FetchGroup fg{&sm.bar[0], 0u};
    if (lane == 0) { mbar_init(fg.bar, 1); fence_mbar_init(); }
    __syncwarp();
    fg.issue2(lane, sm.raw, in + (uint64_t)iw.x * 128, rec_bytes16<RW>(iw.w & 127u), sm.src[0], in + (uint64_t)iw.y * 128, rec_bytes16<RW>(min(32u, iw.w >> 7)));
    uint32_t buf = 0;

    for (; item < n_items; item += step) {
        const uint32_t n_t = iw.w & 127u, n_s = iw.w >> 7;
        const char* sin = in + (uint64_t)iw.y * 128;
        char* tout = out + (uint64_t)iw.z * 128;
        const bool has_next = item + step < n_items;
        uint4 iw_next = iw;
        if (has_next) iw_next = __ldg(reinterpret_cast<const uint4*>(items) + item + step);
        fg.wait();                    // this item's targets and first source round
        // the lane's own two targets (lane, lane + 32): table entries; bounding box of the whole item
        const bool vA = lane < n_t, vB = lane + 32 < n_t;
        double ft[3] = {0.0, 0.0, 0.0};      // slots: the frame of the targets' side (the sources' is re-read per round: registers)
        if constexpr (SLOTS) {
#pragma unroll
            for (int d = 0; d < 3; ++d) ft[d] = __ldg(item_frames + 6 * (size_t)item + d);
        }
        float4 oA = make_float4(0.f, 0.f, 0.f, 0.f), oB = oA;      // x, y, z, 4 h^2
        float hA = 0.f, hB = 0.f;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const uint32_t t = lane + 32 * k;
            float4 p0 = make_float4(0.f, 0.f, 0.f, 0.f), p1 = p0, p2 = make_float4(0.f, 0.f, 1.f, 0.f);
            if (t < n_t) {
                const float* r = sm.raw + RW * t;
                const float h = r[3 + O], rho = r[5 + O], ih = rcp_fast(h);
                p0 = make_float4(rec_x<SLOTS>(r, 0, ft), rec_x<SLOTS>(r, 1, ft), rec_x<SLOTS>(r, 2, ft), 4.0f * h * h);
                p1 = make_float4(r[7 + O], r[8 + O], r[9 + O], r[12 + O]);
                p2 = make_float4(ih, kInvPi * (ih * ih) * (ih * ih), rho, r[11 + O] * rcp_fast(fmaf(h * r[6 + O], rcp_fast(3.0f * rho), 1.0f) * rho * rho));
                if (k == 0) hA = h; else hB = h;
                if constexpr (SWITCH) sm.tB[t] = balsara(r);
            }
            sm.t0[t] = p0; sm.t1[t] = p1; sm.t2[t] = p2;
            if (k == 0) oA = p0; else oB = p0;
        }
        __syncwarp();                 // every lane has read its records: sm.raw becomes the result area
        for (uint32_t v = lane; v < 80; v += 32) reinterpret_cast<float4*>(sm.raw)[v] = make_float4(0.f, 0.f, 0.f, 0.f);
        const float reach_t = 2.0f * warp_max_pos(fmaxf(hA, hB));
        const float lox = warp_min(vB ? fminf(oA.x, oB.x) : oA.x, vA), hix = warp_max(vB ? fmaxf(oA.x, oB.x) : oA.x, vA);
        const float loy = warp_min(vB ? fminf(oA.y, oB.y) : oA.y, vA), hiy = warp_max(vB ? fmaxf(oA.y, oB.y) : oA.y, vA);
        const float loz = warp_min(vB ? fminf(oA.z, oB.z) : oA.z, vA), hiz = warp_max(vB ? fmaxf(oA.z, oB.z) : oA.z, vA);
        const float ri2_max = warp_max_pos(fmaxf(fmaf(oA.x, oA.x, fmaf(oA.y, oA.y, oA.z * oA.z)), fmaf(oB.x, oB.x, fmaf(oB.y, oB.y, oB.z * oB.z))));
        float tile_hc2 = 0.f, tile_b2 = 0.f;      // over the tile being filled: largest (2 h_j)^2, largest |s|^2 (warp-uniform)
        __syncwarp();

        auto flush = [&](uint32_t cnt) {
            // cut-off of a target against this tile: max((2 h_i)^2, largest (2 h_j)^2 in the tile) -- a superset of max(2h_i, 2h_j) per pair.
            // Targets that cannot reach the tile's bounding box sit this flush out; the others get a lane (or half of one).
            const Box box = tile_box(sm.f, cnt, lane);
            const bool aA = vA && box_dist2(box, oA.x, oA.y, oA.z) < fmaxf(oA.w, tile_hc2) * kReachSlack;
            const bool aB = vB && box_dist2(box, oB.x, oB.y, oB.z) < fmaxf(oB.w, tile_hc2) * kReachSlack;
            const uint32_t n_act = compact_targets(sm.act, aA, aB, lane, lt);
            const float hc2_tile = tile_hc2, b2 = 3.0f * fmaxf(tile_b2, ri2_max);
            tile_hc2 = 0.f; tile_b2 = 0.f;
            if (n_act == 0) return;
            const bool dual = n_act > 32;                // else: one target per lane, two of its hits per iteration
            const bool wA = lane < n_act, wB = dual && lane + 32 < n_act;
            const uint32_t tA = wA ? sm.act[lane] : 0, tB = wB ? sm.act[lane + 32] : tA;
            const float4 pA = sm.t0[tA], pB = sm.t0[tB];
            const float cutA = fmaxf(pA.w, hc2_tile), cutB = fmaxf(pB.w, hc2_tile);
            const FilterTarget fA = filter_target(pA.x, pA.y, pA.z, wA ? fmaf(pA.x, pA.x, fmaf(pA.y, pA.y, pA.z * pA.z)) - cutA - kFilterEps * (b2 + cutA) : kNever);
            const FilterTarget fB = filter_target(pB.x, pB.y, pB.z, wB ? fmaf(pB.x, pB.x, fmaf(pB.y, pB.y, pB.z * pB.z)) - cutB - kFilterEps * (b2 + cutB) : kNever);
            uint32_t m[4];
            filter_masks(sm.f, cnt, dual, fA, fB, m);
            // Phase 2.  Inside a pair of cells the number of neighbours per target is heavy-tailed (0 .. ~30: targets next to the
            // other cell against targets three layers away), so lanes that walked their own targets' masks would leave most of
            // the warp idle.  Instead
            //   (a) every lane cuts its masks into UNITS (target, <= 4 set bits of one mask word), numbered RANK-major over the
            //       lanes (all first units, then all second units, ...: making the units, and adding up their partial sums,
            //       takes as many warp steps as the busiest lane has units);
            //   (b) the units are evaluated 32 at a time, one per lane, each leaving its partial sums in shared memory;
            //   (c) the lane that made a unit adds its partial sums to the target's running sums, in unit order.
            // Acceleration sums ~60 terms an order of magnitude larger than the result (pressure forces cancel): compensated (Kahan)
            // adds keep the rounding of the running sums out of the 1e-6 max|a| budget.
            // (r01 / early r02 also had a WALK instantiation for large cells -- every lane walking its own two targets' masks; with
            // particles in Morton order inside cells the units win on every workload: eagle-like force 32.6 -> 26.0 ms, configs[4]
            // at 2^23 particles 42.5 -> 39.1 ms per step, configs[2] 3.83 -> 3.44 ms, configs[1] 413 -> 349 us -- so it is gone.)
            const uint32_t cA0 = __popc(m[0]), cA1 = __popc(m[1]), cB0 = __popc(m[2]), cB1 = __popc(m[3]);
            const uint32_t nuA = (cA0 + kUnitBits - 1) / kUnitBits + (cA1 + kUnitBits - 1) / kUnitBits;
            const uint32_t nuB = (cB0 + kUnitBits - 1) / kUnitBits + (cB1 + kUnitBits - 1) / kUnitBits, nu = nuA + nuB;
            float axA = 0.f, ayA = 0.f, azA = 0.f, duA = 0.f, vsA = 0.f, axB = 0.f, ayB = 0.f, azB = 0.f, duB = 0.f, vsB = 0.f;
            {
                const uint32_t max_nu = __reduce_max_sync(kFull, nu);
                __syncwarp();     // the filter has read sm.f: its first bytes now hold the unit list
                uint32_t* upos = reinterpret_cast<uint32_t*>(&sm.f);                        // [kUnitCap] the unit's (up to) four bits of a mask word
                unsigned char* utgt = reinterpret_cast<unsigned char*>(upos + kUnitCap);    // [kUnitCap] the unit's target | tile half << 7
                float4* part_a = reinterpret_cast<float4*>(sm.raw + 320);                   // [kUnitCap] a (3), du
                float* part_v = sm.raw + 320 + 4 * kUnitCap;                                // [kUnitCap] v_sig
                float cxA = 0.f, cyA = 0.f, czA = 0.f, cxB = 0.f, cyB = 0.f, czB = 0.f;
                uint32_t cw = 0, mw = m[0];             // the mask word being cut (0, 1: target A; 2, 3: target B) and what is left of it
                const uint32_t m1 = m[1], m2 = m[2], m3 = m[3];
                for (uint32_t r = 0; r < max_nu;) {
                    // (a) the next ranks, as many as fit into a window of kUnitCap units
                    const uint32_t r0 = r;
                    uint32_t cum = 0;
                    while (r < max_nu) {
                        const uint32_t bal = __ballot_sync(kFull, nu > r), n_r = __popc(bal);
                        if (cum + n_r > (uint32_t)kUnitCap) break;
                        if (nu > r) {
                            while (mw == 0) { ++cw; mw = cw == 1 ? m1 : (cw == 2 ? m2 : m3); }
                            const uint32_t before = mw;
#pragma unroll
                            for (int q = 0; q < kUnitBits; ++q) mw &= ~shr_clamp(0x80000000u, __clz(mw));      // __clz(0) = 32: the shift gives 0, nothing cleared
                            const uint32_t idx = cum + __popc(bal & lt);
                            upos[idx] = before ^ mw;
                            utgt[idx] = (unsigned char)((r < nuA ? tA : tB) | ((cw & 1) << 7));
                        }
                        cum += n_r; ++r;
                    }
                    __syncwarp();

                    // (b) evaluation: both halves of the packed arithmetic serve the unit's target
                    for (uint32_t u0 = 0; u0 < cum; u0 += 32) {
                        const uint32_t u = u0 + lane;
                        const bool valid = u < cum;
                        uint32_t um = valid ? upos[u] : 0u;
                        const uint32_t tw = valid ? utgt[u] : 0u, t = tw & 127u, ebase = (tw >> 7) * kHalf;
                        const float4 P = sm.t0[t], Q = sm.t1[t], S = sm.t2[t];
                        const ForceTargets2 T{dup2(P.x), dup2(P.y), dup2(P.z), dup2(Q.x), dup2(Q.y), dup2(Q.z), dup2(Q.w), dup2(S.x), dup2(S.y), dup2(S.z), dup2(S.w), P.w, P.w, switch_pair<SWITCH>(sm, t, t, true)};
                        u64 ax = 0, ay = 0, az = 0, du = 0;
                        float vsig = 0.f;
                        auto two = [&](uint32_t ja, uint32_t jb) {
                            const ForcePair2 o = force_pair2<SWITCH>(T, K, sm.ta[ja], sm.ta[jb], sm.tb[ja], sm.tb[jb], sm.tc[ja], sm.tc[jb],
                                                                     switch_pair<SWITCH>(sm, ja, jb, false));
                            ax = fma2(o.fr, o.ex, ax); ay = fma2(o.fr, o.ey, ay); az = fma2(o.fr, o.ez, az);
                            du = fma2(o.dg, o.vr, du);
                            vsig = fmaxf(vsig, fmaxf(o.vsa, o.vsb));
                        };
                        // the unit's neighbours two by two; a slot without one points at its half's dummy (entry 32)
#pragma unroll
                        for (uint32_t q = 0; q < kUnitBits; q += 2) {
                            const uint32_t j0 = __clz(um);
                            um &= ~shr_clamp(0x80000000u, j0);
                            const uint32_t j1 = __clz(um);
                            um &= ~shr_clamp(0x80000000u, j1);
                            if (q == 0 || __any_sync(kFull, j0 != 32u)) two(ebase + j0, ebase + j1);
                        }
                        if (valid) {
                            float ax0, ax1, ay0, ay1, az0, az1, du0, du1;
                            unpack2(ax, ax0, ax1); unpack2(ay, ay0, ay1); unpack2(az, az0, az1); unpack2(du, du0, du1);
                            part_a[u] = make_float4(ax0 + ax1, ay0 + ay1, az0 + az1, du0 + du1);
                            part_v[u] = vsig;
                        }
                    }
                    __syncwarp();

                    // (c) partial sums -> the targets' running sums
                    uint32_t c2 = 0;
                    for (uint32_t q = r0; q < r; ++q) {
                        const uint32_t bal = __ballot_sync(kFull, nu > q);
                        if (nu > q) {
                            const uint32_t idx = c2 + __popc(bal & lt);
                            const float4 pa = part_a[idx];
                            const float pv = part_v[idx];
                            float y, t;
                            if (q < nuA) {
                                y = pa.x + cxA; t = axA + y; cxA = y - (t - axA); axA = t;      // c holds minus the error so far
                                y = pa.y + cyA; t = ayA + y; cyA = y - (t - ayA); ayA = t;
                                y = pa.z + czA; t = azA + y; czA = y - (t - azA); azA = t;
                                duA += pa.w; vsA = fmaxf(vsA, pv);
                            } else {
                                y = pa.x + cxB; t = axB + y; cxB = y - (t - axB); axB = t;
                                y = pa.y + cyB; t = ayB + y; cyB = y - (t - ayB); ayB = t;
                                y = pa.z + czB; t = azB + y; czB = y - (t - azB); azB = t;
                                duB += pa.w; vsB = fmaxf(vsB, pv);
                            }
                        }
                        c2 += __popc(bal);
                    }
                    __syncwarp();     // the unit list and the partial sums are rewritten by the next window / flush
                }
            }
            if (wA) { float* o = sm.raw + 5 * tA; o[0] += axA; o[1] += ayA; o[2] += azA; o[3] += duA; o[4] = fmaxf(o[4], vsA); }
            if (wB) { float* o = sm.raw + 5 * tB; o[0] += axB; o[1] += ayB; o[2] += azB; o[3] += duB; o[4] = fmaxf(o[4], vsB); }
        };

        uint32_t cnt = 0;
        const uint32_t n_rounds = max(1u, (n_s + 31) >> 5);
        for (uint32_t r = 0; r <= n_rounds; ++r) {      // round n_rounds: the closing flush (one flush site: code size)
            float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a, c = a;
            float s2 = 0.f;
            bool ok = false;
            uint32_t ball = 0, n_ok = 0;
            if (r < n_rounds) {
                const uint32_t j0 = 32 * r, nj = min(32u, n_s - j0);
                if (r > 0) fg.wait();
                // one step ahead: the next round of this item (the next item's records are fetched once the results have left sm.raw)
                if (r + 1 < n_rounds) fg.issue1(lane, sm.src[buf ^ 1], sin + (uint64_t)(j0 + 32) * (RW * 4), rec_bytes16<RW>(min(32u, n_s - j0 - 32)));
                if (lane < nj) {
                    const float* rec = sm.src[buf] + RW * lane;
                    const float h = rec[3 + O], rho = rec[5 + O];
                    double fs[3] = {0.0, 0.0, 0.0};
                    if constexpr (SLOTS) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) fs[d] = __ldg(item_frames + 6 * (size_t)item + 3 + d);
                    }
                    const float reach = fmaxf(reach_t, 2.0f * h) * kReachSlack;
                    a = make_float4(rec_x<SLOTS>(rec, 0, fs), rec_x<SLOTS>(rec, 1, fs), rec_x<SLOTS>(rec, 2, fs), 4.0f * h * h);
                    ok = a.x > lox - reach && a.x < hix + reach && a.y > loy - reach && a.y < hiy + reach && a.z > loz - reach && a.z < hiz + reach;
                    if (ok) {
                        b = make_float4(rec[7 + O], rec[8 + O], rec[9 + O], rec[4 + O]);
                        c = make_float4(rho, rec[11 + O] * rcp_fast(fmaf(h * rec[6 + O], rcp_fast(3.0f * rho), 1.0f) * rho * rho), rec[12 + O], rcp_fast(h));
                        s2 = fmaf(a.x, a.x, fmaf(a.y, a.y, a.z * a.z));
                    }
                }
                ball = __ballot_sync(kFull, ok); n_ok = __popc(ball);
            }
            if (cnt + n_ok > kTile || (r == n_rounds && cnt)) { flush(cnt); __syncwarp(); cnt = 0; }
            if (r < n_rounds) {
                if (ok) {
                    const uint32_t pos = cnt + __popc(ball & lt), e = pos + (pos >> 5);      // half * 33 + index in the half
                    sm.ta[e] = a; sm.tb[e] = b; sm.tc[e] = c;
                    if constexpr (SWITCH) sm.sB[e] = balsara(sm.src[buf] + RW * lane);
                    filter_put(sm.f, pos, a.x, a.y, a.z, s2);
                }
                tile_hc2 = fmaxf(tile_hc2, warp_max_pos(ok ? a.w : 0.f));
                tile_b2 = fmaxf(tile_b2, warp_max_pos(s2));
                cnt += n_ok;
                buf ^= 1;
            }
        }
        __syncwarp();
        // the running results are already in FORCE_OUT record layout: they leave as coalesced 16-byte stores
        const uint32_t nvec = (n_t * 5 + 3) >> 2;
        for (uint32_t v = lane; v < nvec; v += 32) reinterpret_cast<uint4*>(tout)[v] = reinterpret_cast<const uint4*>(sm.raw)[v];
        __syncwarp();
        if (has_next) {
            fg.issue2(lane, sm.raw, in + (uint64_t)iw_next.x * 128, rec_bytes16<RW>(iw_next.w & 127u),
                      sm.src[buf], in + (uint64_t)iw_next.y * 128, rec_bytes16<RW>(min(32u, iw_next.w >> 7)));
        }
        iw = iw_next;
    }
}

template <class K>
int32_t loop_grid(K kernel, size_t smem, uint32_t* grid) {
    int sms = 0, per_sm = 0;
    if (int32_t rc = device_sms(&sms)) return rc;
    if (smem > 48 * 1024) SPH_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    SPH_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kLoopWarps * 32, smem));
    *grid = (uint32_t)(sms * max(per_sm, 1));
    return SPH_OK;
}

}  // namespace

int32_t launch_density(const sph_batch* b, const char* d_in, char* d_out, cudaStream_t st) {
    if (b->n_items == 0) return SPH_OK;
    uint32_t full_grid = 0;
    if (int32_t rc = loop_grid(density_kernel<false>, 0, &full_grid)) return rc;
    const uint32_t grid = min((b->n_items + kLoopWarps - 1) / kLoopWarps, full_grid);
    density_kernel<false><<<grid, kLoopWarps * 32, 0, st>>>(b->d_items_density, d_in, d_out, b->n_items, nullptr);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_density_slots(const sph_batch* b, const SlotTables& sl, const char* d_slots, char* d_out, cudaStream_t st) {
    if (b->n_items == 0) return SPH_OK;
    uint32_t full_grid = 0;
    if (int32_t rc = loop_grid(density_kernel<true>, 0, &full_grid)) return rc;
    const uint32_t grid = min((b->n_items + kLoopWarps - 1) / kLoopWarps, full_grid);
    density_kernel<true><<<grid, kLoopWarps * 32, 0, st>>>(sl.d_items, d_slots, d_out, b->n_items, sl.d_item_frames);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_gradient(const sph_batch* b, const char* d_in, char* d_out, cudaStream_t st) {
    if (b->n_items == 0) return SPH_OK;
    uint32_t full_grid = 0;
    constexpr size_t smem = sizeof(GradientWarpSmem) * kLoopWarps;
    if (int32_t rc = loop_grid(gradient_kernel, smem, &full_grid)) return rc;
    const uint32_t grid = min((b->n_items + kLoopWarps - 1) / kLoopWarps, full_grid);
    gradient_kernel<<<grid, kLoopWarps * 32, smem, st>>>(b->d_items_gradient, d_in, d_out, b->n_items);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

template <bool SWITCH, bool SLOTS>
static int32_t launch_force_t(const sph_batch* b, const LoopItem* items, const double* item_frames, const char* d_in, char* d_out, const sph_params& prm, cudaStream_t st) {
    if (b->n_items == 0) return SPH_OK;
    uint32_t full_grid = 0;
    constexpr size_t smem = sizeof(ForceWarpSmemT<SLOTS ? 17 : (SWITCH ? 18 : 13)>) * kLoopWarps;
    if (int32_t rc = loop_grid(force_kernel<SWITCH, SLOTS>, smem, &full_grid)) return rc;
    const uint32_t grid = min((b->n_items + kLoopWarps - 1) / kLoopWarps, full_grid);
    force_kernel<SWITCH, SLOTS><<<grid, kLoopWarps * 32, smem, st>>>(items, d_in, d_out, b->n_items, prm.alpha, prm.beta, item_frames);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_force(const sph_batch* b, const char* d_in, char* d_out, const sph_params& prm, cudaStream_t st) {
    return launch_force_t<false, false>(b, b->d_items_force, nullptr, d_in, d_out, prm, st);
}

int32_t launch_force3(const sph_batch* b, const char* d_in, char* d_out, const sph_params& prm, cudaStream_t st) {
    return launch_force_t<true, false>(b, b->d_items_force3, nullptr, d_in, d_out, prm, st);
}

int32_t launch_force_slots(const sph_batch* b, const SlotTables& sl, const char* d_slots, char* d_out, const sph_params& prm, cudaStream_t st) {
    return launch_force_t<false, true>(b, sl.d_items, sl.d_item_frames, d_slots, d_out, prm, st);
}

}  // namespace sph
