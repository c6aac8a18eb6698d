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
#define LV_T_CAP 224
#endif
#ifndef LV_T_MINBLOCKS
#define LV_T_MINBLOCKS 5
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
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "LV_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t"
        "@p bra LV_DONE_%=;\n\t"
        "bra LV_WAIT_%=;\n\t"
        "LV_DONE_%=:\n\t}"
        ::"r"(bar), "r"(parity), "r"(200000u) : "memory");     // suspend-time hint (ns): sleep, do not spin
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

// ---- producer / consumer pipeline ------------------------------------------------------
// A block is two independent PAIRS of warps.  Both warps of a pair own the same window of 32
// consecutive sorted slots: the PRODUCER warp forms the tiles, computes the stencil rows, and
// issues the bulk copies into a ring of kTDepth shared-memory slots (one JOB = one round of
// one row batch of one (tile, grid)); the CONSUMER warp waits on a slot's `full` mbarrier
// (armed with the byte count of the copies), walks it and hands it back through the slot's
// `empty` mbarrier.  The latency of the offset loads and of the copies is the producer's; the
// consumer only computes.
#ifndef LV_T_DEPTH
#define LV_T_DEPTH 2
#endif
constexpr int kTDepth = LV_T_DEPTH;
constexpr int kJobFirst = 1;      // first job of a tile: the consumer closes the previous tile
constexpr int kJobEnd = 2;        // no more tiles in this window

struct JobMeta {
    int flags;
    int pair_ab;        // a0 * LV_MAX_TYPES + b
    int clen;           // pairs staged in this slot
    int cpad;           // clen rounded up to the walk step (dummies behind clen)
    int selfbase;       // own pair of a target = selfbase + (its slot >> 1); < -2^28: not in this job
    int first_slot, cnt;
    int nblank;
    float tgt[3 * 32];  // x, y, z of the tile's targets (cnt entries each)
    int blank[64];      // halves outside their run: 2 * pair position + half
};
static_assert(sizeof(JobMeta) % 32 == 0, "slot data must stay 32-byte aligned");

struct RingSlot {
    PairSlot data[kTBuf];
    JobMeta meta;
};

constexpr int kNoSelf = -(1 << 29);

template <bool kCharged, int S>
__global__ void __launch_bounds__(kTThreads, LV_T_MINBLOCKS)
k_pair_force_t(const __grid_constant__ LvDev P, const float4 *__restrict__ pos,
               const float *__restrict__ posP, const uint32_t *__restrict__ off,
               float4 *__restrict__ force)
{
    constexpr int T = TileCfg<S>::T, U = TileCfg<S>::U, kStep = TileCfg<S>::kStep;
    constexpr int kPairs = kTWarps / 2;
    extern __shared__ __align__(32) unsigned char s_raw[];
    RingSlot *s_ring = reinterpret_cast<RingSlot *>(s_raw);                     // [kPairs][kTDepth]
    LvPair *s_pair = reinterpret_cast<LvPair *>(s_ring + kPairs * kTDepth);     // [64]
    unsigned long long *s_bar = reinterpret_cast<unsigned long long *>(s_pair + LV_MAX_TYPES * LV_MAX_TYPES);
    int8_t *s_w = reinterpret_cast<int8_t *>(s_bar + kPairs * kTDepth * 2);     // full[], empty[] per pair

    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int pr_id = wib >> 1;
    const bool producer = (wib & 1) == 0;
    for (int t = threadIdx.x; t < LV_MAX_TYPES * LV_MAX_TYPES; t += kTThreads) {
        s_pair[t] = P.pair[t];
        s_w[t] = P.w[t];
    }
    if (threadIdx.x < kPairs * kTDepth * 2) mbar_init(smem_u32(s_bar + threadIdx.x), 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();

    // the pair's 32 consecutive sorted slots, taken from the END of the sorted order first
    // (the types with the longest ranges sit there)
    const int base = P.n - 32 * (int)(blockIdx.x * kPairs + pr_id + 1);
    if (base + 32 <= 0) return;
    RingSlot *ring = s_ring + pr_id * kTDepth;
    const uint32_t bar_full = smem_u32(s_bar + pr_id * kTDepth * 2);
    const uint32_t bar_empty = bar_full + 8u * kTDepth;
    const int rt = lane % T, rs = lane / T;           // consumer role: target of the tile, sub-stream

    if (producer) {
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
        int job = 0;                                  // jobs emitted: ring slot job % depth
        // wait until the consumer has handed the slot of job `job` back
        auto acquire = [&]() -> RingSlot * {
            const int sl = job % kTDepth, use = job / kTDepth;
            if (use > 0) mbar_wait(bar_empty + 8u * sl, (uint32_t)(use - 1) & 1u);
            // the consumer's (and our own earlier) generic writes to the slot come before the
            // bulk copies that overwrite it
            fence_proxy_async_smem();
            return ring + sl;
        };
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

            const int srcl = t0 + min(lane, cnt - 1);     // lane k holds target k (the last, beyond cnt)
            const float tx = __shfl_sync(kFull, pl.x, srcl);
            const float ty = __shfl_sync(kFull, pl.y, srcl);
            const float tz = __shfl_sync(kFull, pl.z, srcl);
            const int first_slot = base + t0;
            const float bx0 = warp_min(tx), bx1 = warp_max(tx);       // bounding box of the targets
            const float by0 = warp_min(ty), by1 = warp_max(ty);
            const float bz0 = warp_min(tz), bz1 = warp_max(tz);
            bool first = true;
            LV_TSTAT(0, 1);
            LV_TSTAT(7, cnt);
            // header of a job: flags, tile, targets (first job of the tile only)
            auto put_header = [&](RingSlot *sl, int pair_ab, int clen, int cpad, int selfbase) {
                if (lane == 0) {
                    sl->meta.flags = first ? kJobFirst : 0;
                    sl->meta.pair_ab = pair_ab;
                    sl->meta.clen = clen;
                    sl->meta.cpad = cpad;
                    sl->meta.selfbase = selfbase;
                    sl->meta.first_slot = first_slot;
                    sl->meta.cnt = cnt;
                }
                if (first && lane < cnt) {
                    sl->meta.tgt[lane] = tx;
                    sl->meta.tgt[32 + lane] = ty;
                    sl->meta.tgt[64 + lane] = tz;
                }
            };
            for (int b = 0; b < P.n_types; ++b) {
                LV_TSTAT(1, 1);
                const int w = (int)s_w[a0 * LV_MAX_TYPES + b];
                const float rc2 = s_pair[a0 * LV_MAX_TYPES + b].rc2;
                const LvGridDev g = P.grid[b];
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
                const float rct2 = rc2 * 1.0009765625f * (g.inv_h * g.inv_h);

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
                    // ---- the runs as aligned slot pairs, end to end
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
                    // the targets' own slots (b = a only) lie in the run of the tile's row: stream
                    // position of pair q of the sorted order = selfbase + q
                    int selfbase = kNoSelf;
                    if (b == a0) {
                        const unsigned own = __ballot_sync(kFull, js <= (uint32_t)first_slot && (uint32_t)first_slot < je);
                        if (own) selfbase = __shfl_sync(kFull, pre - pj, __ffs(own) - 1);
                    }
                    for (int c0 = 0; c0 < total; c0 += kTCap) {
                        const int clen = min(kTCap, total - c0);
                        const int cpad = (clen + kStep - 1) / kStep * kStep;
                        LV_TSTAT(5, cpad / S);
                        LV_TSTAT(6, 1);
                        RingSlot *sl = acquire();
                        put_header(sl, a0 * LV_MAX_TYPES + b, clen, cpad, selfbase == kNoSelf ? kNoSelf : selfbase - c0);
                        // halves outside their run: before an odd js, after an odd je
                        const int last = pre + len - 1;
                        const bool bf = len > 0 && (js & 1u) && pre >= c0 && pre < c0 + clen;
                        const bool bl = len > 0 && (je & 1u) && last >= c0 && last < c0 + clen;
                        const unsigned mf = __ballot_sync(kFull, bf), ml = __ballot_sync(kFull, bl);
                        const unsigned lt = (1u << lane) - 1u;
                        if (bf) sl->meta.blank[__popc(mf & lt)] = 2 * (pre - c0);
                        if (bl) sl->meta.blank[__popc(mf) + __popc(ml & lt)] = 2 * (last - c0) + 1;
                        if (lane == 0) sl->meta.nblank = __popc(mf) + __popc(ml);
                        // pad the last walk iteration with far dummies (never in range)
                        if (clen + lane < cpad) {
                            float4 *d = reinterpret_cast<float4 *>(sl->data + clen + lane);
                            d[0] = make_float4(1e18f, 1e18f, 0.f, 0.f);
                            d[1] = make_float4(0.f, 0.f, 0.f, 0.f);
                        }
                        __syncwarp();
                        const uint32_t fb = bar_full + 8u * (uint32_t)(job % kTDepth);
                        const int lo_ = max(pre, c0), hi_ = min(pre + len, c0 + clen);
                        if (hi_ > lo_)
                            bulk_g2s(smem_u32(sl->data + (lo_ - c0)), posP + 8 * (size_t)(pj + (lo_ - pre)),
                                     32u * (uint32_t)(hi_ - lo_), fb);
                        if (lane == 0) mbar_arrive_expect_tx(fb, 32u * (uint32_t)clen);
                        first = false;
                        ++job;
                    }
                }
            }
            if (first) {          // a tile without a single candidate: an empty job carries it
                RingSlot *sl = acquire();
                put_header(sl, a0 * LV_MAX_TYPES, 0, 0, kNoSelf);
                if (lane == 0) sl->meta.nblank = 0;
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_full + 8u * (uint32_t)(job % kTDepth));
                ++job;
            }
        }
        RingSlot *sl = acquire();
        if (lane == 0) {
            sl->meta.flags = kJobEnd;
            mbar_arrive(bar_full + 8u * (uint32_t)(job % kTDepth));
        }
        return;
    }

    // ---- consumer: walk the staged jobs of the pair's window in order
    f32x2 fx2 = 0ull, fy2 = 0ull, fz2 = 0ull;         // (0.f, 0.f): partial sums of the two halves
    f32x2 tx2 = 0ull, ty2 = 0ull, tz2 = 0ull;
    int nin = 0, my_slot = 0, t_first = 0, t_cnt = 0;
    bool have = false;
    for (int job = 0;; ++job) {
        RingSlot *sl = ring + job % kTDepth;
        mbar_wait(bar_full + 8u * (uint32_t)(job % kTDepth), (uint32_t)(job / kTDepth) & 1u);
        const int flags = sl->meta.flags;
        if (flags & (kJobFirst | kJobEnd)) {
            if (have) {
                // close the previous tile: the two halves, then the S partial sums of every target
                // (fixed order); one writer per target
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
                if (rs == 0 && rt < t_cnt) force[t_first + rt] = make_float4(fx, fy, fz, __int_as_float(nin));
            }
            if (flags & kJobEnd) break;
            have = true;
            fx2 = fy2 = fz2 = 0ull;
            nin = 0;
            t_first = sl->meta.first_slot;
            t_cnt = sl->meta.cnt;
            const int k = min(rt, t_cnt - 1);          // lanes beyond the tile mirror its last target
            const float tx = sl->meta.tgt[k], ty = sl->meta.tgt[32 + k], tz = sl->meta.tgt[64 + k];
            tx2 = pack2(tx, tx); ty2 = pack2(ty, ty); tz2 = pack2(tz, tz);
            my_slot = t_first + k;
        }
        const int cpad = sl->meta.cpad, nblank = sl->meta.nblank, selfbase = sl->meta.selfbase;
        const LvPair pr = s_pair[sl->meta.pair_ab];
        const f32x2 c12v = pack2(pr.c12, pr.c12), nc6v = pack2(-pr.c6, -pr.c6), qqv = pack2(pr.qq, pr.qq);
        // blank the halves that lie outside their run (the copies have landed)
        for (int k = lane; k < nblank; k += 32) {
            const int e = sl->meta.blank[k];
            (&sl->data[e >> 1].x0)[e & 1] = 1e18f;
        }
        __syncwarp();
        // ---- walk: lane (rt, rs) takes pair positions rs, rs + S, ...
        const bool self_here = selfbase > kNoSelf / 2;
        const int sp = selfbase + (my_slot >> 1) - rs;     // own pair: p0 + u S == sp
        const int sq0 = (!self_here || (my_slot & 1)) ? kNoSelf : sp;     // ... and own half
        const int sq1 = (self_here && (my_slot & 1)) ? sp : kNoSelf;
        const uint32_t q = smem_u32(sl->data) + 32u * (uint32_t)rs;
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
        if (self_here) walk(IntC<1>());
        else walk(IntC<0>());
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8u * (uint32_t)(job % kTDepth));
    }
}

constexpr size_t kTSmem = (size_t)(kTWarps / 2) * kTDepth * sizeof(RingSlot) +
                          LV_MAX_TYPES * LV_MAX_TYPES * sizeof(LvPair) +
                          (size_t)(kTWarps / 2) * kTDepth * 2 * sizeof(unsigned long long) +
                          LV_MAX_TYPES * LV_MAX_TYPES;

template <bool kCharged, int S>
cudaError_t launch_tile(const LvDev &P, const LvBufs &B, cudaStream_t st)
{
    const int per_block = 32 * (kTWarps / 2);
    const int blocks = (P.n + per_block - 1) / per_block;
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
