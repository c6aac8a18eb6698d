// lv_internal.cuh -- private to csrc/: device parameter block, buffer table and
// the launch wrappers shared by lv_api.cu, lv_kernels.cu and lv_sort.cu.
// Nothing here is seen by the oracle (oracle/ shares no code with this tree).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "lv.h"

// {r_c^2, 48 eps sigma^12, 24 eps sigma^6, k_C q_a q_b} of one type pair, fp32,
// rounded once from fp64 (include/lv.h: lv_set_types).
struct LvPair {
    float rc2, c12, c6, qq;
};

struct LvTypeDev {
    float dt_over_m;  // dt / m_a
    float a, b;       // velocity retention and kick std (R11, R15)
    float mass;
    float radius;     // r_a = sigma_a / 2
    float pad0, pad1, pad2;
};

struct LvGridDev {
    float lo, inv_h;
    int32_t G;
    uint32_t base;
};

// Passed BY VALUE to every kernel (__grid_constant__): lives in the constant
// bank of the launch, so several lv_sim handles never share mutable state.
struct LvDev {
    int32_t n, n_types;
    uint32_t n_cells;
    int32_t wall_mode;
    LvPair pair[LV_MAX_TYPES * LV_MAX_TYPES];
    LvTypeDev type[LV_MAX_TYPES];
    LvGridDev grid[LV_MAX_TYPES];
    int8_t w[LV_MAX_TYPES * LV_MAX_TYPES];
    int8_t wl[LV_MAX_TYPES * LV_MAX_TYPES];   // stencil half-widths for r_c,ab + skin (list build)
    float dt, g;
    float om2[3];
    int32_t sched_mode;
    int64_t sched_steps;
    double R0, R1;
    double wall_k_d[LV_MAX_TYPES];
    double radius_d[LV_MAX_TYPES];
    uint32_t seed_lo, seed_hi;
    uint32_t n_scan_tiles;   // tiles of the cell-count scan (counting sort)
    // skin neighbour list (lv_set_neighbour_list); list_cap = 0: off
    int32_t list_cap;        // != 0: list on
    uint32_t list_pool;      // pool of the list in entries (4 bytes each)
    uint32_t n_list_tiles;   // tiles of the scan over the list lengths
    int32_t list_lanes_forced;   // LV_OPT_LIST_LANES: 0 = chosen on the device
    float skin;              // list radius = r_c,ab + skin
    float half_skin2;        // rebuild when an NP has moved farther than this (squared) since the build
    // LV_FORCE_TILE: a target of type a more than this many cells of its grid along x from a
    // tile's first target starts a new tile
    int32_t tile_cells[LV_MAX_TYPES];
};

// Device-resident scalars.
struct LvDevState {
    long long step;        // index of the next step to take
    unsigned int status;   // LV_ST_* bits, sticky
    unsigned int ticket;   // blocks of k_update that have read `step`
    // skin list: rebuild[n & 1] != 0 -> step n rebuilds the cell structures and the list.
    // The update of step n raises rebuild[(n + 1) & 1] and, once every block has read
    // rebuild[n & 1], clears it for step n + 2.
    unsigned int rebuild[2];
    unsigned int n_rebuilds;   // rebuilds since lv_set_state
    // skin list: 1 = the list of the last rebuild fits the pool and is in use; 0 = the pool was
    // too small at the last count -- steps rebuild the cells and use the cell kernel until a
    // later count (every 64th step) fits again
    unsigned int list_ok;
    unsigned int list_lanes;       // lanes that share one NP's list in the force kernel (8, 16 or 32)
    unsigned int n_fallback;       // steps taken on the cell kernel since lv_set_state
    // 1 after lv_set_state: the first step runs on the cell kernel and the list is built at the
    // second -- a list pays only if steps follow (set_state / step(1) / get_state loops)
    unsigned int list_defer;
    unsigned long long list_total; // entries counted by the count pass that is under way
    unsigned long long list_used;  // entries the last build reserved
    // 1: list_len[] holds the lengths of a valid list in the present slot order, so the next
    // rebuild can size the new lists from them and fill in ONE walk
    unsigned int list_prev;
    // raised during a rebuild when the one-walk build cannot be used or a list outgrew its
    // reserve: the exact two-pass build (count, scan, fill) of the same step takes over
    unsigned int list_redo;
    unsigned int n_exact;          // rebuilds done by the exact two-pass build since lv_set_state
    unsigned int pad;
    unsigned long long list_true;  // true (padded) entries of the list being filled / last filled
};

struct LvBufs {
    float4 *posA, *velA;   // current state, slot order of the last rebuild (w: type / id bits)
    float4 *posB, *velB;   // cell-sorted copy of the current step
    float4 *force;         // pair force per sorted slot (w: in-range count bits)
    // key_in: cell key per current slot.  Radix mode: val_in = slot, key_out / val_out =
    // sorted keys / permutation.  Counting mode: val_in = arrival rank inside the cell,
    // key_out = per-cell slot lists in arrival order, val_out = permutation.
    uint32_t *key_in, *key_out, *val_in, *val_out;
    uint32_t *cell_off;    // [n_cells + 1]
    uint32_t *cell_cnt;    // [n_cells + 1] NPs per cell; zero between steps (counting mode)
    unsigned long long *scan_tile;   // [n_scan_tiles] look-back words of the scan
    unsigned int *scan_ticket;
    void *sort_temp;
    size_t sort_temp_bytes;
    LvDevState *st;
    unsigned char *staging;  // n * 28 bytes: host<->device state transfers
    // Pair-interleaved copy of posB for the packed force kernel: slots 2p and 2p+1 share
    // 32 bytes {x0, x1, y0, y1, z0, z1, w0, w1}; slots n .. 2*ceil(n/2)+1 are dummies far
    // outside every cut-off.  Written by the gather only when that kernel is selected.
    float *posP;
    // skin neighbour list: the NP at sorted slot i owns list[list_start[i] .. list_start[i + 1]),
    // its neighbours' slots in walk order, padded to a multiple of 4 entries with the dummy slot n (posA[n] = posB[n]: far outside every cut-off);
    // list_cnt = padded lengths (input of the scan, zero between builds), list_start = their
    // exclusive scan; pos_ref = positions at the last build.
    uint32_t *list;
    uint32_t *list_cnt;      // [n + 1] reserved lengths (input of the scan, zero between builds)
    uint32_t *list_start;    // [n + 1]
    uint32_t *list_len;      // [n] true lengths, padded to a multiple of 4
    unsigned long long *list_scan_tile;
    unsigned int *list_scan_ticket;
    float4 *pos_ref;
};

// droplet radius after n steps (step (iii)); fp64 on host and device
__host__ __device__ inline double lv_radius_of(int mode, double R0, double R1, long long S, long long n)
{
    if (mode == LV_SCHED_CONST || S <= 0) return R0;
    long long m = n < 0 ? 0 : (n > S ? S : n);
    if (m == S) return R1;
    double f = (double)m / (double)S;
    if (mode == LV_SCHED_LINEAR) return R0 + (R1 - R0) * f;
    return sqrt(R0 * R0 + (R1 * R1 - R0 * R0) * f);
}

#ifndef LV_SCAN_TILE
#define LV_SCAN_TILE 8192
#endif
constexpr int kScanTile = LV_SCAN_TILE;   // cells per tile of the cell-count scan

// ---- launch wrappers (lv_kernels.cu) -- all asynchronous on `st` ----------
cudaError_t lvk_hash(const LvDev &P, const LvBufs &B, cudaStream_t st);
cudaError_t lvk_bounds_scatter(const LvDev &P, const LvBufs &B, bool packed, cudaStream_t st);
// counting sort (one radix digit = the whole key): hash + count, scan, place, rank + gather
// guarded = true (skin-list steps): the kernel returns at once unless this step rebuilds
cudaError_t lvk_hash_count(const LvDev &P, const LvBufs &B, bool guarded, cudaStream_t st);
cudaError_t lvk_scan_cells(const LvDev &P, const LvBufs &B, bool guarded, cudaStream_t st);
cudaError_t lvk_place(const LvDev &P, const LvBufs &B, bool guarded, cudaStream_t st);
cudaError_t lvk_rank_gather(const LvDev &P, const LvBufs &B, bool packed, bool guarded, cudaStream_t st);
// skin list: build from the cell structures (guarded), force from the list, update in list order
// count (rows per warp) -> scan (tile offsets, pool check) -> fill, all guarded
cudaError_t lvk_list_build(const LvDev &P, const LvBufs &B, cudaStream_t st);
// sets the condition of the graph's IF node (the rebuild chain) from this step's rebuild flag
cudaError_t lvk_list_cond(unsigned long long handle, const LvBufs &B, cudaStream_t st);
// cell kernel of a list step: runs only while the list does not fit its pool
cudaError_t lvk_pair_force_fallback(const LvDev &P, const LvBufs &B, cudaStream_t st);
cudaError_t lvk_pair_force_list(const LvDev &P, const LvBufs &B, cudaStream_t st);
cudaError_t lvk_update_list(const LvDev &P, const LvBufs &B, cudaStream_t st);
cudaError_t lvk_keys_sorted(const LvDev &P, const LvBufs &B, uint32_t *out, cudaStream_t st);
cudaError_t lvk_pair_force(const LvDev &P, const LvBufs &B, int variant, cudaStream_t st);
// shared-candidate-stream kernel (lv_force_tile.cu): `substreams` lanes per target (1 .. 32, a
// power of two); lvk_tile_prepare raises its shared-memory limit (call once, outside capture)
cudaError_t lvk_tile_prepare();
cudaError_t lvk_pair_force_tile(const LvDev &P, const LvBufs &B, int substreams, bool charged, cudaStream_t st);
bool lvk_any_charge(const LvDev &P);
// hash_next: also hash + histogram the new positions for the next step's counting sort
cudaError_t lvk_update(const LvDev &P, const LvBufs &B, bool hash_next, cudaStream_t st);
cudaError_t lvk_pack_state(const LvDev &P, const LvBufs &B, const float *pos, const float *vel,
                           const int32_t *type, long long step, cudaStream_t st);
cudaError_t lvk_unpack_state(const LvDev &P, const LvBufs &B, float *pos, float *vel,
                             int32_t *type, cudaStream_t st);
// order_b: `force` is in the slot order of B (ids in velB), else of A (ids in velA)
cudaError_t lvk_unpack_forces(const LvDev &P, const LvBufs &B, bool order_b, float *force,
                              int32_t *count, cudaStream_t st);
cudaError_t lvk_ids_sorted(const LvDev &P, const LvBufs &B, uint32_t *ids, cudaStream_t st);

// ---- sort (lv_sort.cu): stable LSD radix sort of (key, val) over end_bit bits
size_t lvs_temp_bytes(int n, int end_bit);
cudaError_t lvs_sort_pairs(void *temp, size_t temp_bytes, const uint32_t *key_in, uint32_t *key_out,
                           const uint32_t *val_in, uint32_t *val_out, int n, int end_bit,
                           cudaStream_t st);

// observables (lv_observe_*): integer histograms + fp64 sums into caller-zeroed device memory;
// h_grid = cell edge per type grid (host)
cudaError_t lvk_rdf_hist(const LvDev &P, const LvBufs &B, const double *h_grid, double dr, int n_bins,
                         unsigned long long *hist, cudaStream_t st);
cudaError_t lvk_radial_hist(const LvDev &P, const LvBufs &B, const double *h_grid, double R, double dr,
                            int n_bins, unsigned long long *hist, double *sums, cudaStream_t st);

// aggregates: rb2 = T x T squared bond lengths (fp32, host); scratch 3 uint32[n] (device)
cudaError_t lvk_clusters(const LvDev &P, const LvBufs &B, const float *rb2, const double *h_grid,
                         uint32_t *scratch, int32_t *label_by_id, unsigned long long *stats,
                         cudaStream_t st);

// headless perspective view: zbuf W*H u64 (device scratch), rgba W*H u32 (device)
cudaError_t lvk_render(const LvDev &P, const LvBufs &B, const lv_view *view, const float *rot9,
                       double R, unsigned long long *zbuf, uint32_t *rgba, cudaStream_t st);
cudaError_t lvk_render_surface(const LvDev &P, const LvBufs &B, const lv_surface_map *map, double R,
                               const float *tab_dev, unsigned long long *zbuf, uint32_t *rgba,
                               cudaStream_t st);

// FP32 FMA throughput probe (lv_measure_fp32_peak)
cudaError_t lvk_fma_peak(float *scratch, int blocks, int iters, double *flops, cudaStream_t st);
