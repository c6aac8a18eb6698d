// lv_force_tile.cu -- A6 (step ii) as a SHARED-CANDIDATE-STREAM kernel for
// dense states (LV_FORCE_TILE).
//
// The per-lane walk of k_pair_force_s (lv_kernels.cu) has two floors that belong to "one
// lane, one target, its own candidate stream": every warp request gathers 32 distinct
// 16-byte candidates (>= 4 wavefronts of the L1 data pipe) and every candidate costs the
// lane its own run bookkeeping.  Here a warp owns a TILE of T = 32 / S consecutive
// cell-sorted targets of one type (same (y, z) row of their own grid, x spread bounded) and
// S lanes work for each target:
//   rows    -- per neighbour grid b, the lanes of the warp each take one (y, z) row of the
//              union stencil: gap of the row to the tile's bounding box (cell units of
//              grid b, from the contract-#1 coordinates), rows out of reach dropped, the
//              others trimmed to the x cells the cut-off sphere around the box can reach
//              (block-level ball trimming).  A row is ONE contiguous, 16-byte aligned run
//              of float4 slots [off[row + xa], off[row + xb + 1]).
//   stage   -- a warp prefix sum places the runs end to end in the warp's shared-memory
//              buffer; every lane issues a 1-D bulk copy (TMA, cp.async.bulk) of its own
//              run, completion counted in bytes on the warp's mbarrier.
//   walk    -- all lanes walk the SAME staged stream: lane (target t, sub-stream s) reads
//              candidates s, s + S, ... -- T lanes read one address (broadcast), a warp
//              request touches S consecutive float4 (one wavefront for S <= 8); contract #2
//              exactly as everywhere else, the force under a select.
//   reduce  -- the S partial sums of a target are added by xor shuffles in a fixed order
//              (deterministic), one lane per target writes (F, in-range count).
// The target's own slot sits in the stream when b = a; it is rejected by its stream
// position (the tile's targets are consecutive slots of one run), not by r = 0, so a
// coincident pair of distinct NPs still produces the non-finite force of reading R6.
#include "lv_internal.cuh"
#include "lv_device.cuh"

namespace {

constexpr int kTThreads = 128;                 // 4 independent warps
constexpr int kTWarps = kTThreads / 32;
#ifndef LV_T_CAP
#define LV_T_CAP 368
#endif
constexpr int kTCap = LV_T_CAP;                // candidate PAIRS per round of a warp's buffer
constexpr int kTBuf = kTCap + 32;              // + dummy padding of the last walk iteration

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "LV_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra LV_DONE_%=;\n\t"
        "bra LV_WAIT_%=;\n\t"
        "LV_DONE_%=:\n\t}"
        ::"r"(bar), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared (TMA): dst, src 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// order-preserving map float -> uint32 (for redux min / max); NaN sorts to an end, which
// only widens the tile's box
__device__ __forceinline__ uint32_t f2ord(float f)
{
    const uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(uint32_t u)
{
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}
__device__ __forceinline__ float warp_min(float v) { return ord2f(__reduce_min_sync(kFull, f2ord(v))); }
__device__ __forceinline__ float warp_max(float v) { return ord2f(__reduce_max_sync(kFull, f2ord(v))); }

// lower bound (cell units, >= 0) of the distance along one axis between any target of a
// tile spanning [tlo, thi] and any NP binned into cell c: cells c >= 1 have a true lower
// edge and cells c <= G - 2 a true upper edge (the clamp of contract #1 only lengthens the
// two end cells outwards)
__device__ __forceinline__ float axis_gap(int c, float tlo, float thi, int G, float marg)
{
    float g = 0.0f;
    if (c >= 1 && thi < (float)c) g = (float)c - thi;
    else if (c <= G - 2 && tlo > (float)(c + 1)) g = tlo - (float)(c + 1);
    return fmaxf(g - marg, 0.0f);
}

// Counting build (-DLV_T_STATS): tiles, (tile, grid) jobs, row batches, non-empty runs, staged
// candidates, walk iterations x 32 lanes, buffer rounds; read by lv_debug_tile_stats.
#ifdef LV_T_STATS
__device__ unsigned long long g_tstats[8];
#define LV_TSTAT(k, v) do { const unsigned long long v_ = (unsigned long long)(v); if (lane == 0) atomicAdd(&g_tstats[k], v_); } while (0)
#else
#define LV_TSTAT(k, v) do { } while (0)
#endif

// in = r2 < rc2 (and, when the stream holds the target itself, pos != own position): fp32
// contract #2.  count += in; f = in ? f : 0 -- a select, so the NaN / inf of a rejected
// candidate never propagates.  One block so that the count is a single predicated add.
template <bool kSelf>
__device__ __forceinline__ void gate(float r2, float rc2, int pos, int own, float &f, int &count)
{
    if (kSelf)
        asm("{\n\t.reg .pred p;\n\tsetp.lt.f32 p, %2, %3;\n\tsetp.ne.and.s32 p, %4, %5, p;\n\t"
            "@p add.s32 %1, %1, 1;\n\tselp.f32 %0, %0, 0f00000000, p;\n\t}"
            : "+f"(f), "+r"(count) : "f"(r2), "f"(rc2), "r"(pos), "r"(own));
    else
        asm("{\n\t.reg .pred p;\n\tsetp.lt.f32 p, %2, %3;\n\t"
            "@p add.s32 %1, %1, 1;\n\tselp.f32 %0, %0, 0f00000000, p;\n\t}"
            : "+f"(f), "+r"(count) : "f"(r2), "f"(rc2));
}

template <int S> struct TileCfg {
    static constexpr int T = 32 / S;                 // targets per tile
    static constexpr int U = S <= 8 ? 2 : 1;         // candidate PAIRS per lane and walk iteration
    static constexpr int kStep = S * U;              // pair positions per walk iteration
};

// The staged stream is made of ALIGNED SLOT PAIRS of the pair-interleaved copy of the sorted
// positions (LvBufs::posP: 32 bytes {x0, x1, y0, y1, z0, z1, w0, w1} per pair), so that one
// LDS.128 + one LDS.64 hand a lane two candidates already laid out as f32x2 operands
// (FADD2 / FMUL2 / FFMA2: one issue slot for two candidates).  A run [js, je) is staged as
// the pairs [js >> 1, (je + 1) >> 1); the half before an odd js and the half after an odd je
// belong to neighbouring cells and are blanked in shared memory once the copy has landed
// (they are candidates of their own runs, if of any).
struct PairSlot {
    float x0, x1, y0, y1, z0, z1, w0, w1;
};

template <bool kCharged, int S>
__global__ void __launch_bounds__(kTThreads, 4)
k_pair_force_t(const __grid_constant__ LvDev P, const float4 *__restrict__ pos,
               const float *__restrict__ posP, const uint32_t *__restrict__ off,
               float4 *__restrict__ force)
{
    constexpr int T = TileCfg<S>::T, U = TileCfg<S>::U, kStep = TileCfg<S>::kStep;
    extern __shared__ __align__(32) unsigned char s_raw[];
    PairSlot *s_buf = reinterpret_cast<PairSlot *>(s_raw);                      // [kTWarps][kTBuf]
    LvPair *s_pair = reinterpret_cast<LvPair *>(s_buf + kTWarps * kTBuf);       // [64]
    unsigned long long *s_bar = reinterpret_cast<unsigned long long *>(s_pair + LV_MAX_TYPES * LV_MAX_TYPES);
    int8_t *s_w = reinterpret_cast<int8_t *>(s_bar + kTWarps);

    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    for (int t = threadIdx.x; t < LV_MAX_TYPES * LV_MAX_TYPES; t += kTThreads) {
        s_pair[t] = P.pair[t];
        s_w[t] = P.w[t];
    }
    if (threadIdx.x < kTWarps) mbar_init(smem_u32(s_bar + threadIdx.x), 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();

    // the warp's 32 consecutive sorted slots, taken from the END of the sorted order first
    // (the types with the longest ranges sit there)
    const int base = P.n - 32 * (int)(blockIdx.x * kTWarps + wib + 1);
    if (base + 32 <= 0) return;
    const int slot = base + lane;
    const bool live = slot >= 0;
    const float4 pl = pos[live ? slot : 0];
    const int al = live ? __float_as_int(pl.w) : -1;
    int cxl = 0, cyl = 0, czl = 0;
    if (live) {
        const LvGridDev ga = P.grid[al];
        cxl = cell_coord(pl.x, ga.lo, ga.inv_h, ga.G);
        cyl = cell_coord(pl.y, ga.lo, ga.inv_h, ga.G);
        czl = cell_coord(pl.z, ga.lo, ga.inv_h, ga.G);
    }
    PairSlot *buf = s_buf + wib * kTBuf;
    const uint32_t buf_u32 = smem_u32(buf), bar = smem_u32(s_bar + wib);
    uint32_t phase = 0u;
    const int rt = lane % T, rs = lane / T;           // role: target of the tile, sub-stream

    unsigned todo = __ballot_sync(kFull, live);
    while (todo) {
        // ---- tile: up to T consecutive lanes of one type in one (y, z) row of their grid, at
        // most tile_cells cells along x from the first (the slots are sorted by cell, not by x)
        const int t0 = __ffs(todo) - 1;
        const int a0 = __shfl_sync(kFull, al, t0);
        const int cx0 = __shfl_sync(kFull, cxl, t0);
        const int cy0 = __shfl_sync(kFull, cyl, t0), cz0 = __shfl_sync(kFull, czl, t0);
        const bool same = live && lane >= t0 && al == a0 && cyl == cy0 && czl == cz0 &&
                          (unsigned)(cxl - cx0) <= (unsigned)P.tile_cells[a0];
        const unsigned run = __ballot_sync(kFull, same) >> t0;      // bit 0 = lane t0 (set)
        int cnt = __ffs(~run) - 1;                                  // leading run of ones
        if (cnt < 0 || cnt > T) cnt = T;                            // ~run == 0: all 32 lanes
        cnt = min(cnt, 32 - t0);
        todo &= ~((cnt >= 32 ? 0xffffffffu : ((1u << cnt) - 1u)) << t0);

        const int srcl = t0 + min(rt, cnt - 1);       // lanes beyond the tile mirror its last target
        const float tx = __shfl_sync(kFull, pl.x, srcl);
        const float ty = __shfl_sync(kFull, pl.y, srcl);
        const float tz = __shfl_sync(kFull, pl.z, srcl);
        const int first_slot = base + t0;
        const int my_slot = base + srcl;
        // bounding box of the tile's targets
        const float bx0 = warp_min(tx), bx1 = warp_max(tx);
        const float by0 = warp_min(ty), by1 = warp_max(ty);
        const float bz0 = warp_min(tz), bz1 = warp_max(tz);
        const f32x2 tx2 = pack2(tx, tx), ty2 = pack2(ty, ty), tz2 = pack2(tz, tz);

        f32x2 fx2 = 0ull, fy2 = 0ull, fz2 = 0ull;     // (0.f, 0.f): partial sums of the two halves
        int nin = 0;
        LV_TSTAT(0, 1);
        LV_TSTAT(7, cnt);
        for (int b = 0; b < P.n_types; ++b) {
            LV_TSTAT(1, 1);
            const int w = (int)s_w[a0 * LV_MAX_TYPES + b];
            const LvPair pr = s_pair[a0 * LV_MAX_TYPES + b];
            const LvGridDev g = P.grid[b];
            const f32x2 c12v = pack2(pr.c12, pr.c12), nc6v = pack2(-pr.c6, -pr.c6), qqv = pack2(pr.qq, pr.qq);
            // the box on grid b in contract-#1 coordinates (the expression is monotone in x, so
            // these are the extremes of the targets' own coordinates)
            const float txlo = __fmul_rn(__fsub_rn(bx0, g.lo), g.inv_h), txhi = __fmul_rn(__fsub_rn(bx1, g.lo), g.inv_h);
            const float tylo = __fmul_rn(__fsub_rn(by0, g.lo), g.inv_h), tyhi = __fmul_rn(__fsub_rn(by1, g.lo), g.inv_h);
            const float tzlo = __fmul_rn(__fsub_rn(bz0, g.lo), g.inv_h), tzhi = __fmul_rn(__fsub_rn(bz1, g.lo), g.inv_h);
            const int ya = cell_coord(by0, g.lo, g.inv_h, g.G) - w, yb = cell_coord(by1, g.lo, g.inv_h, g.G) + w;
            const int za = cell_coord(bz0, g.lo, g.inv_h, g.G) - w, zb = cell_coord(bz1, g.lo, g.inv_h, g.G) + w;
            const int ny = yb - ya + 1, nrows = ny * (zb - za + 1);
            const float inv_ny = 1.0f / (float)ny;
            // cell units: rounding of contract #1 moves t by < (G + 8) 2^-23; 4x that as margin
            const float marg = (float)(g.G + 8) * 4.76837158e-7f;
            const float rct2 = pr.rc2 * 1.0009765625f * (g.inv_h * g.inv_h);

            for (int r0 = 0; r0 < nrows; r0 += 32) {
                // ---- rows: one (y, z) row of the union stencil per lane
                const int r = r0 + lane;
                int iz = (int)(((float)r + 0.5f) * inv_ny), iy = r - iz * ny;
                if (iy < 0) { --iz; iy += ny; }
                if (iy >= ny) { ++iz; iy -= ny; }
                const int y = ya + iy, z = za + iz;
                bool ok = r < nrows && (unsigned)y < (unsigned)g.G && (unsigned)z < (unsigned)g.G;
                const float gy = axis_gap(y, tylo, tyhi, g.G, marg), gz = axis_gap(z, tzlo, tzhi, g.G, marg);
                const float rem = rct2 - gy * gy - gz * gz;
                ok = ok && rem > 1e-6f;
                const float remp = fmaxf(rem, 1e-6f);
                const float xh = fmaf(remp, rsqrt_approx(remp), marg);       // sqrt to 2 ulp, inside marg
                // cells 0 and G - 1 are open outwards: clamp the range into the grid
                const int xa = max(0, min(__float2int_rd(txlo - xh), g.G - 1));
                const int xb = min(g.G - 1, max(__float2int_rd(txhi + xh), 0));
                uint32_t js = 0u, je = 0u;
                if (ok) {
                    const uint32_t rowb = g.base + (uint32_t)((z * g.G + y) * g.G);
                    js = __ldg(off + rowb + xa);
                    je = __ldg(off + rowb + xb + 1);
                }
                // ---- stage: the runs as aligned slot pairs, end to end
                const int pj = (int)(js >> 1);
                const int len = je > js ? (int)((je + 1u) >> 1) - pj : 0;      // pairs
                int inc = len;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const int v = __shfl_up_sync(kFull, inc, d);
                    if (lane >= d) inc += v;
                }
                const int total = __shfl_sync(kFull, inc, 31);
                LV_TSTAT(2, 1);
                LV_TSTAT(3, __popc(__ballot_sync(kFull, len > 0)));
                LV_TSTAT(4, total);
                if (total == 0) continue;
                const int pre = inc - len;
                // the target's own slot (b = a only): the run of the tile's row holds every target
                // of the tile; own pair position and half, relative to the stream of this batch
                int self_pair = -1 - 2 * kTCap;
                if (b == a0) {
                    const unsigned own = __ballot_sync(kFull, js <= (uint32_t)first_slot && (uint32_t)first_slot < je);
                    if (own) {
                        const int o = __ffs(own) - 1;
                        self_pair = __shfl_sync(kFull, pre - pj, o) + (my_slot >> 1);
                    }
                }
                for (int c0 = 0; c0 < total; c0 += kTCap) {
                    const int clen = min(kTCap, total - c0);
                    // every lane has left the previous walk; order its generic accesses to the
                    // buffer before the bulk copies that overwrite it
                    __syncwarp();
                    fence_proxy_async_smem();
                    const int lo_ = max(pre, c0), hi_ = min(pre + len, c0 + clen);
                    if (hi_ > lo_)
                        bulk_g2s(buf_u32 + 32u * (uint32_t)(lo_ - c0), posP + 8 * (size_t)(pj + (lo_ - pre)),
                                 32u * (uint32_t)(hi_ - lo_), bar);
                    if (lane == 0) mbar_arrive_expect_tx(bar, 32u * (uint32_t)clen);
                    // pad the last walk iteration with far dummies (never in range)
                    const int cpad = (clen + kStep - 1) / kStep * kStep;
                    LV_TSTAT(5, cpad / S);
                    LV_TSTAT(6, 1);
                    if (clen + lane < cpad) {
                        float4 *d = reinterpret_cast<float4 *>(buf + clen + lane);
                        d[0] = make_float4(1e18f, 1e18f, 0.f, 0.f);
                        d[1] = make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                    mbar_wait(bar, phase);
                    phase ^= 1u;
                    // blank the halves outside the run: before an odd js, after an odd je
                    if (len > 0) {
                        if ((js & 1u) && pre >= c0 && pre < c0 + clen) buf[pre - c0].x0 = 1e18f;
                        const int last = pre + len - 1;
                        if ((je & 1u) && last >= c0 && last < c0 + clen) buf[last - c0].x1 = 1e18f;
                    }
                    __syncwarp();
                    // ---- walk: lane (rt, rs) takes pair positions rs, rs + S, ...
                    const int sp = self_pair - c0 - rs;            // own pair: p0 + u S == sp
                    const int sq0 = (my_slot & 1) ? -1 - 2 * kTCap : sp;     // ... and own half
                    const int sq1 = (my_slot & 1) ? sp : -1 - 2 * kTCap;
                    const uint32_t q = buf_u32 + 32u * (uint32_t)rs;
                    auto walk = [&](auto self_c) {
                        constexpr bool kSelf = decltype(self_c)::value != 0;
#pragma unroll 2
                        for (int p0 = 0; p0 < cpad; p0 += kStep) {
                            f32x2 X[U], Y[U], Z[U];
#pragma unroll
                            for (int u = 0; u < U; ++u) {
                                const uint32_t ad = q + 32u * (uint32_t)(p0 + u * S);
                                asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(X[u]), "=l"(Y[u]) : "r"(ad));
                                asm volatile("ld.shared.b64 %0, [%1+16];" : "=l"(Z[u]) : "r"(ad));
                            }
#pragma unroll
                            for (int u = 0; u < U; ++u) {
                                const f32x2 dx = sub2(tx2, X[u]), dy = sub2(ty2, Y[u]), dz = sub2(tz2, Z[u]);
                                const f32x2 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));   // contract #2, per half
                                float r2a, r2b;
                                unpack2(r2, r2a, r2b);
                                const f32x2 rinv = pack2(rsqrt_approx(r2a), rsqrt_approx(r2b));
                                const f32x2 ir2 = mul2(rinv, rinv);
                                const f32x2 ir6 = mul2(mul2(ir2, ir2), ir2);
                                f32x2 f = mul2(fma2(c12v, ir6, nc6v), ir6);
                                if (kCharged) f = fma2(qqv, rinv, f);
                                f = mul2(f, ir2);
                                float fa, fb;
                                unpack2(f, fa, fb);
                                gate<kSelf>(r2a, pr.rc2, p0 + u * S, sq0, fa, nin);
                                gate<kSelf>(r2b, pr.rc2, p0 + u * S, sq1, fb, nin);
                                f = pack2(fa, fb);
                                fma2_acc(fx2, f, dx);
                                fma2_acc(fy2, f, dy);
                                fma2_acc(fz2, f, dz);
                            }
                        }
                    };
                    if (self_pair >= 0) walk(IntC<1>());
                    else walk(IntC<0>());
                }
            }
        }
        // ---- the two halves, then the S partial sums of every target (fixed order); one
        // writer per target
        float fx, fy, fz, hx, hy, hz;
        unpack2(fx2, fx, hx); fx += hx;
        unpack2(fy2, fy, hy); fy += hy;
        unpack2(fz2, fz, hz); fz += hz;
#pragma unroll
        for (int d = T; d < 32; d <<= 1) {
            fx += __shfl_xor_sync(kFull, fx, d);
            fy += __shfl_xor_sync(kFull, fy, d);
            fz += __shfl_xor_sync(kFull, fz, d);
            nin += __shfl_xor_sync(kFull, nin, d);
        }
        if (rs == 0 && rt < cnt) force[first_slot + rt] = make_float4(fx, fy, fz, __int_as_float(nin));
    }
}

constexpr size_t kTSmem = (size_t)kTWarps * kTBuf * sizeof(PairSlot) + LV_MAX_TYPES * LV_MAX_TYPES * sizeof(LvPair) +
                          kTWarps * sizeof(unsigned long long) + LV_MAX_TYPES * LV_MAX_TYPES;

template <bool kCharged, int S>
cudaError_t launch_tile(const LvDev &P, const LvBufs &B, cudaStream_t st)
{
    const int blocks = (P.n + kTThreads - 1) / kTThreads;
    k_pair_force_t<kCharged, S><<<blocks, kTThreads, kTSmem, st>>>(P, B.posB, B.posP, B.cell_off, B.force);
    return cudaGetLastError();
}

template <bool kCharged, int S>
cudaError_t prepare_tile()
{
    return cudaFuncSetAttribute(k_pair_force_t<kCharged, S>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)kTSmem);
}

}  // namespace

// Raise the dynamic shared-memory limit of every instantiation (once per process and device;
// not a stream operation, so it is called from lv_bind, outside any capture).
cudaError_t lvk_tile_prepare()
{
    cudaError_t e = cudaSuccess;
#define LV_PREP(S)                                                   \
    if (e == cudaSuccess) e = prepare_tile<false, S>();              \
    if (e == cudaSuccess) e = prepare_tile<true, S>();
    LV_PREP(1) LV_PREP(2) LV_PREP(4) LV_PREP(8) LV_PREP(16) LV_PREP(32)
#undef LV_PREP
    return e;
}

#ifdef LV_T_STATS
extern "C" int lv_debug_tile_stats(unsigned long long *out, int reset)
{
    if (out && cudaMemcpyFromSymbol(out, g_tstats, sizeof(g_tstats)) != cudaSuccess) return -1;
    if (reset) {
        unsigned long long z[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        if (cudaMemcpyToSymbol(g_tstats, z, sizeof(z)) != cudaSuccess) return -1;
    }
    return 0;
}
#endif

cudaError_t lvk_pair_force_tile(const LvDev &P, const LvBufs &B, int substreams, bool charged, cudaStream_t st)
{
#define LV_CASE(S)                                                                     \
    case S: return charged ? launch_tile<true, S>(P, B, st) : launch_tile<false, S>(P, B, st);
    switch (substreams) {
        LV_CASE(1) LV_CASE(2) LV_CASE(4) LV_CASE(8) LV_CASE(16) LV_CASE(32)
    default: return cudaErrorInvalidValue;
    }
#undef LV_CASE
}
