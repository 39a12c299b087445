// DENSITY and FORCE interaction loops over cell / cell-pair tasks.
//
// Nothing here is a dense contraction (a few percent of the candidate pairs are neighbours and the per-pair
// work is a distance test), so this is plain FP32 ALU work, not tensor-core work.
//
// One CTA of 128 threads per task.  For each direction (side I gathers from side J, then J from I; a self task
// has one direction) the source records are staged tile by tile in shared memory as float4s, and every thread
// owns one target particle; cells smaller than the CTA are covered by G = 128/TP thread groups that each scan a
// slice of the tile and whose partial sums are combined in a fixed order through shared memory.
#include "internal.h"

namespace sph {

namespace {

constexpr int kLoopThreads = 128;
constexpr int kTile = 256;                 // source particles per shared-memory tile
constexpr float kInvPi = 0.318309886183790671538f;

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

struct Dir { uint32_t tgt, src; };

__global__ void __launch_bounds__(kLoopThreads)
density_kernel(const SideRec* __restrict__ sides, const uint32_t* __restrict__ task_side0, const uint32_t* __restrict__ task_order,
               const uint32_t* __restrict__ off_in, const uint32_t* __restrict__ off_out, const char* __restrict__ in,
               char* __restrict__ out, uint32_t n_tasks) {
    __shared__ float4 s_src[kTile];                 // x, y, z, m
    __shared__ float s_part[4][kLoopThreads];
    const int tid = threadIdx.x;
    for (uint32_t tt = blockIdx.x; tt < n_tasks; tt += gridDim.x) {
        const uint32_t t = task_order[tt];
        const uint32_t s0 = task_side0[t], ns = task_side0[t + 1] - s0;
        for (uint32_t dir = 0; dir < ns; ++dir) {
            const uint32_t tgt = s0 + dir, src = ns == 1 ? s0 : s0 + 1 - dir;
            const uint32_t n_t = sides[tgt].count, n_s = sides[src].count;
            const float* tin = reinterpret_cast<const float*>(in + (uint64_t)off_in[tgt] * 128);
            const float* sin = reinterpret_cast<const float*>(in + (uint64_t)off_in[src] * 128);
            float4* tout = reinterpret_cast<float4*>(out + (uint64_t)off_out[tgt] * 128);
            const uint32_t tp = n_t <= 32 ? 32 : (n_t <= 64 ? 64 : 128), groups = kLoopThreads / tp;
            const uint32_t il = tid & (tp - 1), grp = tid / tp;
            for (uint32_t i0 = 0; i0 < n_t; i0 += tp) {
                const uint32_t i = i0 + il;
                const bool valid = i < n_t;
                float xi = 0, yi = 0, zi = 0, hi = 0;
                if (valid) { xi = tin[5 * i]; yi = tin[5 * i + 1]; zi = tin[5 * i + 2]; hi = tin[5 * i + 3]; }
                const float hc2 = 4.0f * hi * hi, inv_h = valid ? 1.0f / hi : 0.f;
                const float n3 = kInvPi * inv_h * inv_h * inv_h, n4 = n3 * inv_h;
                float rho = 0, rho_dh = 0, wc = 0, wc_dh = 0;
                for (uint32_t j0 = 0; j0 < n_s; j0 += kTile) {
                    const uint32_t tn = min((uint32_t)kTile, n_s - j0);
                    __syncthreads();
                    for (uint32_t j = tid; j < tn; j += kLoopThreads) {
                        const float* r = sin + 5 * (uint64_t)(j0 + j);
                        s_src[j] = make_float4(r[0], r[1], r[2], r[4]);
                    }
                    __syncthreads();
                    const uint32_t per = (tn + groups - 1) / groups;
                    const uint32_t jb = grp * per, je = min(tn, jb + per);
                    for (uint32_t j = jb; j < je; ++j) {
                        const float4 s = s_src[j];
                        const float dx = xi - s.x, dy = yi - s.y, dz = zi - s.z;
                        const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                        if (r2 < hc2) {
                            const float q = sqrtf(r2) * inv_h;
                            float w, dw;
                            spline(q, &w, &dw);
                            const float wv = w * n3, dv = -fmaf(q, dw, 3.0f * w) * n4;
                            rho = fmaf(s.w, wv, rho); rho_dh = fmaf(s.w, dv, rho_dh);
                            wc += wv; wc_dh += dv;
                        }
                    }
                }
                if (groups > 1) {        // combine the thread groups' partial sums in a fixed order
                    __syncthreads();
                    s_part[0][tid] = rho; s_part[1][tid] = rho_dh; s_part[2][tid] = wc; s_part[3][tid] = wc_dh;
                    __syncthreads();
                    if (grp == 0)
                        for (uint32_t g = 1; g < groups; ++g) {
                            rho += s_part[0][tid + g * tp]; rho_dh += s_part[1][tid + g * tp];
                            wc += s_part[2][tid + g * tp]; wc_dh += s_part[3][tid + g * tp];
                        }
                }
                if (grp == 0 && valid) tout[i] = make_float4(rho, rho_dh, wc, wc_dh);
            }
        }
    }
}

__global__ void __launch_bounds__(kLoopThreads)
force_kernel(const SideRec* __restrict__ sides, const uint32_t* __restrict__ task_side0, const uint32_t* __restrict__ task_order,
             const uint32_t* __restrict__ off_in, const uint32_t* __restrict__ off_out, const char* __restrict__ in,
             char* __restrict__ out, uint32_t n_tasks, float alpha, float beta) {
    __shared__ float4 s_a[kTile];   // x, y, z, 4 h^2
    __shared__ float4 s_b[kTile];   // vx, vy, vz, m
    __shared__ float4 s_c[kTile];   // rho, A = P / (Omega rho^2), c_s, 1/h
    __shared__ float s_part[5][kLoopThreads];
    const int tid = threadIdx.x;
    for (uint32_t tt = blockIdx.x; tt < n_tasks; tt += gridDim.x) {
        const uint32_t t = task_order[tt];
        const uint32_t s0 = task_side0[t], ns = task_side0[t + 1] - s0;
        for (uint32_t dir = 0; dir < ns; ++dir) {
            const uint32_t tgt = s0 + dir, src = ns == 1 ? s0 : s0 + 1 - dir;
            const uint32_t n_t = sides[tgt].count, n_s = sides[src].count;
            const float* tin = reinterpret_cast<const float*>(in + (uint64_t)off_in[tgt] * 128);
            const float* sin = reinterpret_cast<const float*>(in + (uint64_t)off_in[src] * 128);
            float* tout = reinterpret_cast<float*>(out + (uint64_t)off_out[tgt] * 128);
            const uint32_t tp = n_t <= 32 ? 32 : (n_t <= 64 ? 64 : 128), groups = kLoopThreads / tp;
            const uint32_t il = tid & (tp - 1), grp = tid / tp;
            for (uint32_t i0 = 0; i0 < n_t; i0 += tp) {
                const uint32_t i = i0 + il;
                const bool valid = i < n_t;
                // FORCE_IN record: xr0 xr1 xr2 h m rho rho_dh v0 v1 v2 u P cs
                float xi = 0, yi = 0, zi = 0, hi = 1, rhoi = 1, rho_dhi = 0, vxi = 0, vyi = 0, vzi = 0, Pi = 0, ci = 0;
                if (valid) {
                    const float* r = tin + 13 * (uint64_t)i;
                    xi = r[0]; yi = r[1]; zi = r[2]; hi = r[3]; rhoi = r[5]; rho_dhi = r[6]; vxi = r[7]; vyi = r[8]; vzi = r[9]; Pi = r[11]; ci = r[12];
                }
                const float hc2i = valid ? 4.0f * hi * hi : 0.f, inv_hi = 1.0f / hi;
                const float n4i = kInvPi * (inv_hi * inv_hi) * (inv_hi * inv_hi);
                const float Ai = Pi / ((1.0f + hi * rho_dhi / (3.0f * rhoi)) * rhoi * rhoi);
                float ax = 0, ay = 0, az = 0, du = 0, vsig = 0;
                for (uint32_t j0 = 0; j0 < n_s; j0 += kTile) {
                    const uint32_t tn = min((uint32_t)kTile, n_s - j0);
                    __syncthreads();
                    for (uint32_t j = tid; j < tn; j += kLoopThreads) {
                        const float* r = sin + 13 * (uint64_t)(j0 + j);
                        const float h = r[3], rho = r[5];
                        s_a[j] = make_float4(r[0], r[1], r[2], 4.0f * h * h);
                        s_b[j] = make_float4(r[7], r[8], r[9], r[4]);
                        s_c[j] = make_float4(rho, r[11] / ((1.0f + h * r[6] / (3.0f * rho)) * rho * rho), r[12], 1.0f / h);
                    }
                    __syncthreads();
                    const uint32_t per = (tn + groups - 1) / groups;
                    const uint32_t jb = grp * per, je = min(tn, jb + per);
                    for (uint32_t j = jb; j < je; ++j) {
                        const float4 a = s_a[j];
                        const float dx = xi - a.x, dy = yi - a.y, dz = zi - a.z;
                        const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                        if (r2 < fmaxf(hc2i, valid ? a.w : 0.f) && r2 > 0.f) {
                            const float4 b = s_b[j], c = s_c[j];
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
                    }
                }
                if (groups > 1) {
                    __syncthreads();
                    s_part[0][tid] = ax; s_part[1][tid] = ay; s_part[2][tid] = az; s_part[3][tid] = du; s_part[4][tid] = vsig;
                    __syncthreads();
                    if (grp == 0)
                        for (uint32_t g = 1; g < groups; ++g) {
                            ax += s_part[0][tid + g * tp]; ay += s_part[1][tid + g * tp]; az += s_part[2][tid + g * tp];
                            du += s_part[3][tid + g * tp]; vsig = fmaxf(vsig, s_part[4][tid + g * tp]);
                        }
                }
                if (grp == 0 && valid) {
                    float* o = tout + 5 * (uint64_t)i;
                    o[0] = ax; o[1] = ay; o[2] = az; o[3] = du; o[4] = vsig;
                }
            }
        }
    }
}

int32_t loop_grid(uint32_t n_tasks, uint32_t* grid) {
    int dev = 0, sms = 0;
    SPH_CUDA_TRY(cudaGetDevice(&dev));
    SPH_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    *grid = min(n_tasks, (uint32_t)sms * 16);
    return SPH_OK;
}

}  // namespace

int32_t launch_density(const sph_batch* b, const uint32_t* d_off_in, const uint32_t* d_off_out, const char* d_in, char* d_out, cudaStream_t st) {
    uint32_t grid = 0;
    if (int32_t rc = loop_grid((uint32_t)b->n_tasks, &grid)) return rc;
    density_kernel<<<grid, kLoopThreads, 0, st>>>(b->d_sides, b->d_task_side0, b->d_task_order, d_off_in, d_off_out, d_in, d_out, (uint32_t)b->n_tasks);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

int32_t launch_force(const sph_batch* b, const uint32_t* d_off_in, const uint32_t* d_off_out, const char* d_in, char* d_out,
                     const sph_params& prm, cudaStream_t st) {
    uint32_t grid = 0;
    if (int32_t rc = loop_grid((uint32_t)b->n_tasks, &grid)) return rc;
    force_kernel<<<grid, kLoopThreads, 0, st>>>(b->d_sides, b->d_task_side0, b->d_task_order, d_off_in, d_off_out, d_in, d_out,
                                                (uint32_t)b->n_tasks, prm.alpha, prm.beta);
    SPH_CUDA_TRY(cudaGetLastError());
    return SPH_OK;
}

}  // namespace sph
