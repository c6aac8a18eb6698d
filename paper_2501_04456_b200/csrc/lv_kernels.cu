// lv_kernels.cu -- sm_100a kernels of the Langevin droplet step.
//
// Rows of SURVEY.md sec. 8(a) / DESIGN.md "Kernels":
//   A2 k_hash            cell key of every NP                       (step i)
//   A4+A5 k_bounds_scatter  cell offsets + gather into cell order
//   A6 k_pair_force      LJ + Coulomb, truncated, unshifted         (step ii)
//   A1+A7 k_update       radius, surface spring, gravity, centrifugal, drag,
//                        Philox kick, new v and x                   (iii-vi)
// A3 (the sort) is in lv_sort.cu.  State layout: float4 pos = (x, y, z, type
// bits), float4 vel = (vx, vy, vz, id bits), 16-byte aligned SoA.
#include "lv_internal.cuh"

namespace {

constexpr int kThreads = 128;

__device__ __forceinline__ int cell_coord(float x, float lo, float inv_h, int G)
{
    // fp32 contract #1: t = fl(fl(x - lo) * inv_h), clamp(floor t), NaN -> 0
    float t = __fmul_rn(__fsub_rn(x, lo), inv_h);
    float f = floorf(t);
    if (!(f >= 0.0f)) return 0;
    if (f > (float)(G - 1)) return G - 1;
    return (int)f;
}

// ---------------------------------------------------------------- A2 hash
__global__ void __launch_bounds__(kThreads)
k_hash(const __grid_constant__ LvDev P, const float4 *__restrict__ pos,
       uint32_t *__restrict__ key, uint32_t *__restrict__ val, LvDevState *st)
{
    int i = blockIdx.x * kThreads + threadIdx.x;
    if (i >= P.n) return;
    float4 p = pos[i];
    int b = __float_as_int(p.w);
    const LvGridDev g = P.grid[b];
    int cx = cell_coord(p.x, g.lo, g.inv_h, g.G);
    int cy = cell_coord(p.y, g.lo, g.inv_h, g.G);
    int cz = cell_coord(p.z, g.lo, g.inv_h, g.G);
    key[i] = g.base + (uint32_t)((cz * g.G + cy) * g.G + cx);
    val[i] = (uint32_t)i;
    float hi = -g.lo;
    bool outside = !(p.x >= g.lo && p.x < hi && p.y >= g.lo && p.y < hi && p.z >= g.lo && p.z < hi);
    if (outside) atomicOr(&st->status, LV_ST_OUTSIDE_GRID);
}

// ------------------------------------------------- A4 + A5 bounds + scatter
// off[c] = first sorted slot whose key is >= c.  Each slot k that starts a new
// key fills off for every cell in (key[k-1], key[k]]; long gaps (empty cells)
// are filled by the whole warp.  No memset of the table is needed.
__device__ __forceinline__ void warp_fill(uint32_t *off, uint32_t first, uint32_t count,
                                          uint32_t value, unsigned lane)
{
    unsigned todo = __ballot_sync(0xffffffffu, count > 0);
    while (todo) {
        int src = __ffs(todo) - 1;
        todo &= todo - 1;
        uint32_t f = __shfl_sync(0xffffffffu, first, src);
        uint32_t c = __shfl_sync(0xffffffffu, count, src);
        uint32_t v = __shfl_sync(0xffffffffu, value, src);
        for (uint32_t t = lane; t < c; t += 32) off[f + t] = v;
    }
}

__global__ void __launch_bounds__(kThreads)
k_bounds_scatter(const __grid_constant__ LvDev P, const uint32_t *__restrict__ key_sorted,
                 const uint32_t *__restrict__ perm, const float4 *__restrict__ posA,
                 const float4 *__restrict__ velA, float4 *__restrict__ posB,
                 float4 *__restrict__ velB, uint32_t *__restrict__ off)
{
    int k = blockIdx.x * kThreads + threadIdx.x;
    unsigned lane = threadIdx.x & 31;
    uint32_t first = 0, count = 0;
    uint32_t tail_first = 0, tail_count = 0;
    if (k < P.n) {
        uint32_t key = key_sorted[k];
        if (k == 0) {
            first = 0; count = key + 1;
        } else {
            uint32_t prev = key_sorted[k - 1];
            first = prev + 1; count = key - prev;
        }
        if (k == P.n - 1) { tail_first = key + 1; tail_count = P.n_cells - key; }
        uint32_t src = perm[k];
        posB[k] = posA[src];
        velB[k] = velA[src];
    }
    warp_fill(off, first, count, (uint32_t)k, lane);
    warp_fill(off, tail_first, tail_count, (uint32_t)P.n, lane);
}

// ------------------------------------------------------------ A6 pair force
__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// One thread per cell-sorted NP.  For every neighbour type b the thread walks
// the (2 w_ab + 1)^2 rows of grid b around its own cell; a row is ONE contiguous
// run of sorted slots [off[first cell], off[last cell + 1]).
__global__ void __launch_bounds__(kThreads)
k_pair_force(const __grid_constant__ LvDev P, const float4 *__restrict__ pos,
             const uint32_t *__restrict__ off, float4 *__restrict__ force)
{
    __shared__ LvPair s_pair[LV_MAX_TYPES * LV_MAX_TYPES];
    if (threadIdx.x < LV_MAX_TYPES * LV_MAX_TYPES) s_pair[threadIdx.x] = P.pair[threadIdx.x];
    __syncthreads();
    int i = blockIdx.x * kThreads + threadIdx.x;
    if (i >= P.n) return;
    const float4 pi = pos[i];
    const int a = __float_as_int(pi.w);
    float fx = 0.f, fy = 0.f, fz = 0.f;
    int cnt = 0;
    for (int b = 0; b < P.n_types; ++b) {
        const LvGridDev g = P.grid[b];
        const int w = P.w[a * LV_MAX_TYPES + b];
        const LvPair pr = s_pair[a * LV_MAX_TYPES + b];
        const int cx = cell_coord(pi.x, g.lo, g.inv_h, g.G);
        const int cy = cell_coord(pi.y, g.lo, g.inv_h, g.G);
        const int cz = cell_coord(pi.z, g.lo, g.inv_h, g.G);
        const int x0 = max(cx - w, 0), x1 = min(cx + w, g.G - 1);
        const int y0 = max(cy - w, 0), y1 = min(cy + w, g.G - 1);
        const int z0 = max(cz - w, 0), z1 = min(cz + w, g.G - 1);
        for (int z = z0; z <= z1; ++z)
            for (int y = y0; y <= y1; ++y) {
                const uint32_t row = g.base + (uint32_t)((z * g.G + y) * g.G);
                const uint32_t js = __ldg(off + row + x0);
                const uint32_t je = __ldg(off + row + x1 + 1);
                for (uint32_t j = js; j < je; ++j) {
                    const float4 pj = __ldg(pos + j);
                    // fp32 contract #2: the in-range predicate, evaluated exactly so
                    const float dx = __fsub_rn(pi.x, pj.x);
                    const float dy = __fsub_rn(pi.y, pj.y);
                    const float dz = __fsub_rn(pi.z, pj.z);
                    const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                    if (r2 < pr.rc2 && j != (uint32_t)i) {
                        const float ir2 = rcp_approx(r2);
                        const float ir6 = ir2 * ir2 * ir2;
                        float f = (pr.c12 * ir6 - pr.c6) * ir6 * ir2;
                        if (pr.qq != 0.0f) f = fmaf(pr.qq * ir2, rsqrt_approx(r2), f);
                        fx = fmaf(f, dx, fx);
                        fy = fmaf(f, dy, fy);
                        fz = fmaf(f, dz, fz);
                        ++cnt;
                    }
                }
            }
    }
    force[i] = make_float4(fx, fy, fz, __int_as_float(cnt));
}

// ------------------------------------------------- A1 + A7 fused update
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__device__ __forceinline__ float u01(uint32_t w)
{
    return ((float)(w >> 9) + 0.5f) * (1.0f / 8388608.0f);   // exact in fp32, in (0, 1)
}

__global__ void __launch_bounds__(kThreads)
k_update(const __grid_constant__ LvDev P, const float4 *__restrict__ posB,
         const float4 *__restrict__ velB, const float4 *__restrict__ force,
         float4 *__restrict__ posA, float4 *__restrict__ velA, LvDevState *st)
{
    int i = blockIdx.x * kThreads + threadIdx.x;
    const long long n = st->step;                      // index of this step
    __syncthreads();
    // the block that takes the last ticket has seen every block read `step`
    if (threadIdx.x == 0 && atomicAdd(&st->ticket, 1u) == gridDim.x - 1) {
        st->ticket = 0u;
        st->step = n + 1;
    }
    if (i >= P.n) return;
    const double Rd = lv_radius_of(P.sched_mode, P.R0, P.R1, P.sched_steps, n + 1);  // (iii), R9
    const float4 p = posB[i];
    const float4 v = velB[i];
    const float4 f = force[i];
    const int a = __float_as_int(p.w);
    const uint32_t id = __float_as_uint(v.w);
    const LvTypeDev ty = P.type[a];

    // (iv) surface spring: pen = |x| - (R - r_a).  |x| ~ 150-250 sigma while pen ~ 0.01 sigma:
    // the difference is taken in fp64 for the NPs near the interface (DESIGN "precision").
    float Fx = f.x, Fy = f.y, Fz = f.z;
    const float rin = (float)Rd - ty.radius;
    const float r2f = fmaf(p.z, p.z, fmaf(p.y, p.y, p.x * p.x));
    const float thr = rin * (1.0f - 1e-5f);
    if (rin <= 0.0f || r2f > thr * thr) {
        const double xd = p.x, yd = p.y, zd = p.z;
        const double r = sqrt(xd * xd + yd * yd + zd * zd);
        const double rad = P.radius_d[a];
        const double pen = r - (Rd - rad);
        if (pen > 0.0 && r > 0.0 && (P.wall_mode == LV_WALL_ONESIDED || pen < 2.0 * rad)) {
            const double s = -P.wall_k_d[a] * pen / r;
            Fx += (float)(s * xd);
            Fy += (float)(s * yd);
            Fz += (float)(s * zd);
        }
    }
    // (v) gravity and centrifugal; drag enters through a
    Fx = fmaf(ty.mass * P.om2[0], p.x, Fx);
    Fy = fmaf(ty.mass * P.om2[1], p.y, Fy);
    Fz = fmaf(ty.mass * P.om2[2], p.z, Fz) - ty.mass * P.g;

    // (vi) Brownian kick: Philox4x32-10 keyed on (seed; id, step), Box-Muller
    float xi0 = 0.f, xi1 = 0.f, xi2 = 0.f;
    if (ty.b != 0.0f) {
        uint32_t w[4];
        philox4x32_10(id, (uint32_t)(unsigned long long)n, (uint32_t)((unsigned long long)n >> 32), 0u,
                      P.seed_lo, P.seed_hi, w);
        const float r01 = sqrtf(-2.0f * logf(u01(w[0])));
        const float r23 = sqrtf(-2.0f * logf(u01(w[2])));
        float s1, c1, s3, c3;
        sincospif(2.0f * u01(w[1]), &s1, &c1);
        sincospif(2.0f * u01(w[3]), &s3, &c3);
        xi0 = r01 * c1; xi1 = r01 * s1; xi2 = r23 * c3;
    }
    const float vx = fmaf(ty.b, xi0, fmaf(ty.dt_over_m, Fx, ty.a * v.x));
    const float vy = fmaf(ty.b, xi1, fmaf(ty.dt_over_m, Fy, ty.a * v.y));
    const float vz = fmaf(ty.b, xi2, fmaf(ty.dt_over_m, Fz, ty.a * v.z));
    const float x = fmaf(P.dt, vx, p.x);
    const float y = fmaf(P.dt, vy, p.y);
    const float z = fmaf(P.dt, vz, p.z);
    posA[i] = make_float4(x, y, z, p.w);
    velA[i] = make_float4(vx, vy, vz, v.w);
    const float chk = (x + y + z) + (vx + vy + vz);
    if (!(fabsf(chk) <= 3.0e38f)) atomicOr(&st->status, LV_ST_NONFINITE);
}

// ------------------------------------------------- state in / out (by id)
__global__ void __launch_bounds__(kThreads)
k_pack_state(int n, const float *__restrict__ pos, const float *__restrict__ vel,
             const int32_t *__restrict__ type, float4 *__restrict__ posA,
             float4 *__restrict__ velA, LvDevState *st, long long step)
{
    int i = blockIdx.x * kThreads + threadIdx.x;
    if (i == 0) { st->step = step; st->status = 0u; st->ticket = 0u; }
    if (i >= n) return;
    posA[i] = make_float4(pos[3 * i], pos[3 * i + 1], pos[3 * i + 2], __int_as_float(type[i]));
    velA[i] = make_float4(vel[3 * i], vel[3 * i + 1], vel[3 * i + 2], __uint_as_float((uint32_t)i));
}

__global__ void __launch_bounds__(kThreads)
k_unpack_state(int n, const float4 *__restrict__ posA, const float4 *__restrict__ velA,
               float *__restrict__ pos, float *__restrict__ vel, int32_t *__restrict__ type)
{
    int i = blockIdx.x * kThreads + threadIdx.x;
    if (i >= n) return;
    const float4 p = posA[i], v = velA[i];
    const uint32_t id = __float_as_uint(v.w);
    if (pos) { pos[3 * id] = p.x; pos[3 * id + 1] = p.y; pos[3 * id + 2] = p.z; }
    if (vel) { vel[3 * id] = v.x; vel[3 * id + 1] = v.y; vel[3 * id + 2] = v.z; }
    if (type) type[id] = __float_as_int(p.w);
}

__global__ void __launch_bounds__(kThreads)
k_unpack_forces(int n, const float4 *__restrict__ force, const float4 *__restrict__ velB,
                float *__restrict__ F, int32_t *__restrict__ count)
{
    int i = blockIdx.x * kThreads + threadIdx.x;
    if (i >= n) return;
    const float4 f = force[i];
    const uint32_t id = __float_as_uint(velB[i].w);
    if (F) { F[3 * id] = f.x; F[3 * id + 1] = f.y; F[3 * id + 2] = f.z; }
    if (count) count[id] = __float_as_int(f.w);
}

__global__ void __launch_bounds__(kThreads)
k_ids_sorted(int n, const float4 *__restrict__ velB, uint32_t *__restrict__ ids)
{
    int i = blockIdx.x * kThreads + threadIdx.x;
    if (i < n) ids[i] = __float_as_uint(velB[i].w);
}

inline int blocks_for(int n) { return n > 0 ? (n + kThreads - 1) / kThreads : 1; }

}  // namespace

cudaError_t lvk_hash(const LvDev &P, const LvBufs &B, cudaStream_t st)
{
    k_hash<<<blocks_for(P.n), kThreads, 0, st>>>(P, B.posA, B.key_in, B.val_in, B.st);
    return cudaGetLastError();
}

cudaError_t lvk_bounds_scatter(const LvDev &P, const LvBufs &B, cudaStream_t st)
{
    k_bounds_scatter<<<blocks_for(P.n), kThreads, 0, st>>>(P, B.key_out, B.val_out, B.posA, B.velA,
                                                           B.posB, B.velB, B.cell_off);
    return cudaGetLastError();
}

cudaError_t lvk_pair_force(const LvDev &P, const LvBufs &B, cudaStream_t st)
{
    k_pair_force<<<blocks_for(P.n), kThreads, 0, st>>>(P, B.posB, B.cell_off, B.force);
    return cudaGetLastError();
}

cudaError_t lvk_update(const LvDev &P, const LvBufs &B, cudaStream_t st)
{
    k_update<<<blocks_for(P.n), kThreads, 0, st>>>(P, B.posB, B.velB, B.force, B.posA, B.velA, B.st);
    return cudaGetLastError();
}

cudaError_t lvk_pack_state(const LvDev &P, const LvBufs &B, const float *pos, const float *vel,
                           const int32_t *type, long long step, cudaStream_t st)
{
    k_pack_state<<<blocks_for(P.n), kThreads, 0, st>>>(P.n, pos, vel, type, B.posA, B.velA, B.st, step);
    return cudaGetLastError();
}

cudaError_t lvk_unpack_state(const LvDev &P, const LvBufs &B, float *pos, float *vel, int32_t *type,
                             cudaStream_t st)
{
    k_unpack_state<<<blocks_for(P.n), kThreads, 0, st>>>(P.n, B.posA, B.velA, pos, vel, type);
    return cudaGetLastError();
}

cudaError_t lvk_unpack_forces(const LvDev &P, const LvBufs &B, float *force, int32_t *count,
                              cudaStream_t st)
{
    k_unpack_forces<<<blocks_for(P.n), kThreads, 0, st>>>(P.n, B.force, B.velB, force, count);
    return cudaGetLastError();
}

cudaError_t lvk_ids_sorted(const LvDev &P, const LvBufs &B, uint32_t *ids, cudaStream_t st)
{
    k_ids_sorted<<<blocks_for(P.n), kThreads, 0, st>>>(P.n, B.velB, ids);
    return cudaGetLastError();
}

// ------------------------------------------------ FP32 FMA peak (measurement aid)
namespace {
__global__ void __launch_bounds__(256) k_fma_peak(float *out, float b, float c, int iters)
{
    float a0 = threadIdx.x * 1e-3f, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f;
    float a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f, a7 = a0 + 7.f;
    for (int k = 0; k < iters; ++k) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fmaf(a0, b, c); a1 = fmaf(a1, b, c); a2 = fmaf(a2, b, c); a3 = fmaf(a3, b, c);
            a4 = fmaf(a4, b, c); a5 = fmaf(a5, b, c); a6 = fmaf(a6, b, c); a7 = fmaf(a7, b, c);
        }
    }
    float s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (s == 12345.678f) out[0] = s;   // never true in practice; keeps the chain alive
}
}  // namespace

cudaError_t lvk_fma_peak(float *scratch, int blocks, int iters, double *flops, cudaStream_t st)
{
    k_fma_peak<<<blocks, 256, 0, st>>>(scratch, 0.999f, 1e-3f, iters);
    *flops = (double)blocks * 256.0 * (double)iters * 64.0 * 2.0;
    return cudaGetLastError();
}
