/*
 * lv.h -- C ABI of the B200-native Langevin droplet step.
 *
 * One data-parallel hot path of the model of Derkachov et al. (arxiv
 * 2501.04456; citations are /root/reference/PAPER.md:<line>): the per-timestep
 * update of N nanoparticles (NPs) of several coexisting types confined in an
 * evaporating or condensing spherical microdroplet, PAPER.md:62-69 (sec. 2.2):
 *   (i)   arrange NPs into cells                         -> hash, sort, cell offsets, scatter
 *   (ii)  Lennard-Jones + Coulomb pair forces in range   -> pair-force kernel
 *   (iii) new droplet radius                             -> schedule, on device
 *   (iv)  surface-tension spring at the interface        \
 *   (v)   gravity, viscosity, centrifugal                 > fused update kernel
 *   (vi)  new velocity and position + Brownian kick      /
 * The formulas (the paper prints none) are the readings R1..R30 of DESIGN.md.
 *
 * Conventions
 *   - Every call returns int: LV_OK (0) or a negative LV_E_* code; nothing is
 *     printed; no C++ exception crosses this boundary.
 *   - "host" / "device" is stated for every pointer.  The caller owns every
 *     buffer it passes; the library owns only the host-side handle and never
 *     allocates device memory (the caller -- torch -- provides one workspace).
 *   - All device work is enqueued on the CUDA stream given to lv_bind and runs
 *     in sm_100a kernels of this library.  There is no CPU fallback.
 *   - State is fp32; tables are derived on the host in fp64 and rounded once.
 *   - Call order: lv_create -> lv_set_types [-> lv_set_forces]
 *     [-> lv_set_droplet_schedule] [-> lv_set_grid] [-> lv_set_option] -> lv_workspace_bytes ->
 *     lv_bind -> lv_set_state -> lv_step / lv_compute_forces / lv_get_* ...
 *     -> lv_destroy.  A setter called after lv_bind returns LV_E_ORDER.
 */
#ifndef LV_H_
#define LV_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LV_MAX_TYPES 8

/* return codes */
#define LV_OK            0
#define LV_E_ARG        -1   /* bad argument */
#define LV_E_ORDER      -2   /* call order violated */
#define LV_E_WORKSPACE  -3   /* workspace too small or misaligned (256 B) */
#define LV_E_CUDA       -4   /* a CUDA runtime call failed; see lv_last_cuda_error */
#define LV_E_NONFINITE  -5   /* sticky: a non-finite position or velocity appeared (R6) */
#define LV_E_NOMEM      -6   /* host allocation failed */
#define LV_E_CAPACITY   -7   /* a size beyond a fixed maximum of the library (lv_observe_rdf_noalloc) */

/* droplet schedule modes: step (iii); radius-square law PAPER.md:58 */
#define LV_SCHED_CONST   0
#define LV_SCHED_LINEAR  1   /* R linear in the step index */
#define LV_SCHED_R2LAW   2   /* R^2 linear in the step index */

/* surface force modes: step (iv) */
#define LV_WALL_ONESIDED 0   /* spring for every pen > 0 (R7) */
#define LV_WALL_WINDOW   1   /* only while 0 < pen < 2 r_NP: the paper's (-r_NP, r_NP) window */

/* status bits (lv_get_status); warnings do not stop the simulation */
#define LV_ST_NONFINITE    1u   /* error: also returned as LV_E_NONFINITE */
#define LV_ST_OUTSIDE_GRID 2u   /* warning: an NP was clamped into a border cell (R22) */
#define LV_ST_LIST_OVERFLOW 4u  /* warning: the skin list did not fit its pool; those steps used the cells */
#define LV_ST_BAD_TYPE     8u   /* error: lv_set_state saw a type outside [0, n_types); that NP was
                                   loaded as type 0 and lv_get_state returns LV_E_ARG */

/* lv_get_debug selectors (parity tests).  The views describe the cell rebuild of the last
 * lv_compute_forces; after lv_step the update kernel has already hashed the NEW positions
 * for the next step (keys, histogram), so only LV_DBG_IDS_SORTED and LV_DBG_GRID are
 * meaningful then. */
#define LV_DBG_KEYS          1  /* uint32[N]   cell key per slot before the sort            */
#define LV_DBG_KEYS_SORTED   2  /* uint32[N]                                                */
#define LV_DBG_PERM          3  /* uint32[N]   sorted slot k came from slot perm[k]         */
#define LV_DBG_CELL_OFFSETS  4  /* uint32[n_cells+1] cell c holds sorted slots [off[c], off[c+1]) */
#define LV_DBG_IDS_SORTED    5  /* uint32[N]   NP id at each sorted slot                    */
#define LV_DBG_GRID          6  /* lv_grid_info (host struct only)                          */

typedef struct lv_sim lv_sim;   /* opaque, host memory, owned by the library */

/* One NP type, PAPER.md:58 ("radius, mass, charge"; per-type spring constant;
 * kick magnitude "passed as a parameter"). */
typedef struct {
    double sigma;    /* NP diameter; r_NP = sigma/2                                   */
    double eps;      /* LJ well depth of the type (used only when eps_TxT == NULL)    */
    double mass;
    double charge;
    double wall_k;   /* surface spring constant                                       */
    double drag_a;   /* velocity retained per step, a = 1 - gamma dt (R11)            */
    double kick_b;   /* std of each component of the random velocity added per step   */
} lv_type;

/* The grids the cell list uses, as exact fp32/fp64 values (LV_DBG_GRID). */
typedef struct {
    int32_t  n_types;
    int32_t  G[LV_MAX_TYPES];           /* cells per axis of the grid of type b        */
    uint32_t base[LV_MAX_TYPES + 1];    /* first key of grid b; base[n_types] = cells  */
    float    lo[LV_MAX_TYPES];          /* lower corner on every axis                  */
    float    inv_h[LV_MAX_TYPES];
    double   h[LV_MAX_TYPES];           /* cell edge                                   */
    int32_t  w[LV_MAX_TYPES * LV_MAX_TYPES]; /* stencil half-width, [a*LV_MAX_TYPES+b] */
} lv_grid_info;

/* a = 1 - gamma dt, b = sqrt((kT/m)(1 - a^2)): explicit Stokes drag and the
 * kick that keeps <v^2> = kT/m stationary (R11, R15).
 * a, b: host, written. */
int lv_langevin_coeffs(double gamma, double kT, double mass, double dt, double *a, double *b);

/* Allocate a handle (host) for n NPs (0 <= n < 2^28) of n_types types (1..LV_MAX_TYPES).
 * seed keys the Philox4x32-10 noise (R15); dt is the time step. */
int lv_create(lv_sim **out, int n, int n_types, uint64_t seed, double dt);

/* NP types and the type x type interaction tables (interactions
 * "within each NP type and between types can be freely set").  All host,
 * copied.  types[n_types].  eps_TxT / sigma_TxT / rcut_TxT: row-major
 * [n_types*n_types] or NULL; NULL -> Lorentz-Berthelot eps_ab = sqrt(eps_a
 * eps_b), sigma_ab = (sigma_a + sigma_b)/2 (= r_A + r_B),
 * r_c,ab = cut_factor * sigma_ab (4 (r_A + r_B) in the paper's
 * runs).  coulomb_k is k_C in U = k_C q_a q_b / r (R5).  Both potentials are
 * truncated at r_c,ab and NOT shifted.  Tables must be
 * symmetric. */
int lv_set_types(lv_sim *s, int n_types, const lv_type *types, const double *eps_TxT,
                 const double *sigma_TxT, const double *rcut_TxT, double cut_factor,
                 double coulomb_k);

/* External fields, step (v) PAPER.md:68: gravity g along -z,
 * centrifugal force m (omega2_xyz[0] x, omega2_xyz[1] y, omega2_xyz[2] z)
 * (isotropic tumbling = (w^2,w^2,w^2); rotation about z = (w^2,w^2,0)), and the
 * surface-force mode.  omega2_xyz: host[3].  Default: 0, (0,0,0), ONESIDED. */
int lv_set_forces(lv_sim *s, double g, const double *omega2_xyz, int wall_mode);

/* Droplet radius as a function of the integer step index n (step (iii),
 * PAPER.md:66): f = min(n, n_steps)/n_steps; CONST R0; LINEAR R0 + (R1-R0) f;
 * R2LAW sqrt(R0^2 + (R1^2-R0^2) f).  R1 > R0 is condensation.
 * During step n the surface stands at R(n+1) (R9). */
int lv_set_droplet_schedule(lv_sim *s, int mode, double R0, double R1, int64_t n_steps);

/* Optional: cells per cut-off k_b >= 1 for the grid of each type (host
 * [n_types]); cell edge h_b = r_c,bb (1 + 2^-9) / k_b.  Default 1. */
int lv_set_grid(lv_sim *s, const int32_t *cells_per_cut);

/* Implementation choices that do not change any result (tests check that):
 *   LV_OPT_SORT          LV_SORT_COUNTING (default): the cell sort as a radix sort
 *                        whose single digit is the whole key -- histogram, scan,
 *                        stable scatter (4 kernels); LV_SORT_RADIX: the on-board
 *                        multi-pass LSD radix sort (CUB) + offsets/scatter kernel.
 *   LV_OPT_FORCE_KERNEL  LV_FORCE_SEGMENTS (default): ball-trimmed stencil rows kept as
 *                        per-lane run lists, walked end to end with the force inline;
 *                        LV_FORCE_PACKED: the same with aligned slot pairs and packed
 *                        f32x2 arithmetic (faster in dense mixed states, slower in
 *                        dilute ones); LV_FORCE_QUEUED: row-by-row lock step with
 *                        per-thread in-range queues; LV_FORCE_SIMPLE: the first kernel.
 *                        The last two are kept as measured baselines.
 *                        LV_FORCE_TILE: shared candidate stream for dense states -- a warp
 *                        owns a tile of 32 / S consecutive sorted targets of one type, the
 *                        stencil rows around the tile's bounding box are staged into shared
 *                        memory by 1-D bulk copies (TMA), and S lanes per target walk the
 *                        same staged stream (steps i-ii).
 *   LV_OPT_TILE_SUBSTREAMS  S of LV_FORCE_TILE: 1, 2, 4 (default), 8, 16 or 32 lanes per target.
 *   LV_OPT_LIST_LANES    lanes that share one NP's neighbour list in the list force kernel:
 *                        1, 2, 4, 8, 16, 32, or 0 (default) = chosen on the device at every
 *                        rebuild from the mean list length.
 *   LV_OPT_TILE_SPAN     cells along x (of the targets' own grid) a tile may extend beyond
 *                        the cell of its first target; -1 (default): cells_per_cut - 1.
 * Every setting gives bit-identical permutations, offsets and neighbour counts;
 * forces agree to rounding. */
#define LV_OPT_SORT          1
#define LV_OPT_FORCE_KERNEL  2
#define LV_SORT_COUNTING     0
#define LV_SORT_RADIX        1
#define LV_FORCE_SIMPLE      0
#define LV_FORCE_QUEUED      1
#define LV_FORCE_SEGMENTS    2
#define LV_FORCE_PACKED      3
#define LV_FORCE_TILE        4
#define LV_OPT_TILE_SUBSTREAMS 3
#define LV_OPT_TILE_SPAN       4
#define LV_OPT_LIST_LANES      5
int lv_set_option(lv_sim *s, int option, int value);

/* Persistent "skin" neighbour list.  The paper rebuilds the cells
 * every step only "to identify which [NPs] are close to each other and can interact"
 * (PAPER.md:64); with capacity != 0 lv_step keeps, per NP, the slots of every NP within
 * r_c,ab + skin at the last rebuild, evaluates the pair force from that list (same fp32
 * contract #2, so the neighbour counts stay bit-identical and the forces agree to rounding),
 * and rebuilds cells + list on the device -- no host round trip -- at the first step after any
 * NP has moved farther than skin/2 from where it was at the build.
 *   skin      length units; <= 0: automatic, 0.16 of the smallest cut-off (needs lv_set_types
 *             first).
 *   capacity  > 0: the list pool holds capacity entries per NP ON AVERAGE (4 * capacity bytes per
 *             NP of workspace; a crowded NP may use more than its share); -1: automatic, 2048
 *             entries per NP but at most 2 GiB, and no list at all below 16 384 NPs (such a
 *             step is bound by launch latency, not by the force kernel); 0 (default): the variant is off and every step
 *             rebuilds the cells, as the paper does.
 * The list is built in two passes (count the lengths, scan them, fill): every NP owns one
 * contiguous run of the pool, and 4 or 8 lanes share an NP in the force kernel (chosen on
 * the device from the mean length).  If a rebuild would need more than the pool, nothing is lost: the
 * warning bit LV_ST_LIST_OVERFLOW is raised and the steps run on the cell kernel (rebuilding the
 * cells every step) until a later count -- taken every 64th step -- fits again.  The choice
 * depends only on the state and the step index, so lv_step(a); lv_step(b) == lv_step(a + b)
 * still holds.  Needs LV_SORT_COUNTING.  lv_compute_forces always uses the cells. */
int lv_set_neighbour_list(lv_sim *s, double skin, int capacity);

/* Cell/list rebuilds since lv_set_state (host int64, written); counts only steps taken
 * with the neighbour list on.  Synchronises. */
int lv_get_rebuild_count(lv_sim *s, int64_t *rebuilds);

/* out6 (host int64[6], written): rebuilds since lv_set_state, list entries the last build
 * reserved, steps taken on the cell kernel because the list did not fit, pool size
 * in entries.  Synchronises. */
int lv_get_list_stats(lv_sim *s, int64_t *out6);

/* Bytes of device workspace lv_bind needs (0 if types are not set). */
size_t lv_workspace_bytes(const lv_sim *s);

/* Freeze the configuration, carve the caller's device workspace (device
 * pointer, 256-byte aligned, >= lv_workspace_bytes, owned by the caller and
 * kept alive until lv_destroy) and remember the CUDA stream (a cudaStream_t
 * passed as void*; NULL = the legacy default stream). */
int lv_bind(lv_sim *s, void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Load a configuration (also the restart path).  pos_xyz,
 * vel_xyz: [n][3] fp32; type: [n] int32 in [0, n_types); all three host
 * (on_device = 0) or all device (on_device = 1); copied.  NP id = row index.
 * step = index of the next step to take.  Synchronises the stream when the
 * sources are host buffers.  A type outside [0, n_types) is loaded as type 0 and raises LV_ST_BAD_TYPE (checked on the
 * device: the call stays asynchronous); lv_get_state then returns LV_E_ARG. */
int lv_set_state(lv_sim *s, const float *pos_xyz, const float *vel_xyz, const int32_t *type,
                 int64_t step, int on_device);

/* Enqueue n full steps on the stream and return without
 * synchronising.  lv_step(a); lv_step(b) equals lv_step(a + b) bit for bit. */
int lv_step(lv_sim *s, int n);

/* Steps (i)-(ii) only on the current state: rebuild the cell structures and
 * compute the pair forces; the state does not change.  Asynchronous. */
int lv_compute_forces(lv_sim *s);

/* Write the state in NP-id order into caller buffers ([n][3] fp32, [n] int32;
 * host or device per on_device; any pointer may be NULL), R = droplet radius
 * R(step) and step (host, may be NULL).  Synchronises the stream.  Returns
 * LV_E_NONFINITE if the sticky error bit is set. */
int lv_get_state(lv_sim *s, float *pos_xyz, float *vel_xyz, int32_t *type, double *R,
                 int64_t *step, int on_device);

/* Pair forces of the last lv_compute_forces / lv_step in NP-id order:
 * force_xyz [n][3] fp32 and neigh_count [n] int32 (NPs inside r_c,ab); host or
 * device per on_device; either may be NULL.  Synchronises. */
int lv_get_forces(lv_sim *s, float *force_xyz, int32_t *neigh_count, int on_device);

/* ---- observables of the paper on the device ----------------
 * Shell index of a distance (fp32 contract #4): (int) fl32(sqrt(r2) * fl32(1/dr))
 * with r2 as in the in-range predicate; counted iff < n_bins (1..8192).  All outputs are host memory, written; any may be NULL.
 * Both calls synchronise the stream and leave the state unchanged.
 *
 * lv_observe_rdf: radial distribution function, Eq. 6.  hist[k] =
 * ordered pairs (i, j != i) whose distance falls in shell k (each NP in turn is the
 * "trial particle"); g[k] = (hist[k]/N) / ((N-1) dV_k / V), dV_k the shell volume and V
 * the droplet volume at the current step; no boundary correction, as printed
 * (PAPER.md:139).  Rebuilds the cell structures of the current state and walks them. */
int lv_observe_rdf(lv_sim *s, double dr, int n_bins, uint64_t *hist, double *g);

/* lv_observe_rdf_noalloc: the same result as lv_observe_rdf (Eq. 6; same
 * kernel, same fp32 contract #4, hist bit-identical) for callers that cannot provide scratch or
 * call an allocator: the histogram scratch of the pair walk is a file-scope device array of
 * the library, LV_NOALLOC_MAX_BINS * 8 bytes = 32 KiB, held by every GPU that loads the library
 * until the process exits (its device address is taken once per device, on the device that is
 * current at the call -- the caller keeps the handle's device current, as for every call).
 * The call makes no cudaMalloc / cudaFree and no host allocation.  n_bins > LV_NOALLOC_MAX_BINS:
 * LV_E_CAPACITY and a line on stderr, nothing launched.  ALL calls of a process share the one
 * array per GPU; it keeps the previous call's counts and is cleared on the handle's stream
 * before the walk.  Two calls that overlap on the GPU (two handles on different streams of one
 * device) RACE on it: serialise them.  hist, g: host memory, written; either may be NULL.
 * Synchronises the stream and leaves the state unchanged. */
#define LV_NOALLOC_MAX_BINS 4096
int lv_observe_rdf_noalloc(lv_sim *s, double dr, int n_bins, uint64_t *hist, double *g);

/* lv_observe_radial: hist[k] = NPs whose distance from the droplet centre falls in shell
 * k and conc[k] = (hist[k]/N) / (dV_k / V), the normalised concentration of Eq. 8
 * (PAPER.md:141); centre[3] = Eq. 4, r_g = Eq. 3, d_f = Eq. 2 solved for D_f with
 * k_f = 1.593 and d_NP the mean NP diameter; n_surf = NPs whose
 * surface lies within one NP radius of the interface, |x| > R - 2 r_a (the NPs that
 * enter Eq. 1). */
int lv_observe_radial(lv_sim *s, double dr, int n_bins, uint64_t *hist, double *conc,
                      double *centre, double *r_g, double *d_f, int64_t *n_surf);

/* lv_observe_clusters: aggregates ("aggregate statistics",
 * "number of sub-aggregates", PAPER.md:58 -- not defined there, reading R23): connected
 * components of the graph whose edges are the pairs with r2 < fl32((bond_factor
 * sigma_ab)^2), r2 as in the in-range predicate.  bond_factor sigma_ab must not exceed
 * r_c,ab (LV_E_ARG).  labels: host int32[n] by NP id, the label of an NP is the smallest
 * NP id of its aggregate; n_clusters, largest (NPs in the largest aggregate), mean_size
 * = n / n_clusters; log2_hist: host uint64[32], aggregates with size in [2^k, 2^(k+1)).
 * All written, any may be NULL.  Rebuilds the cell structures; synchronises; the state
 * does not change. */
int lv_observe_clusters(lv_sim *s, double bond_factor, int32_t *labels, int64_t *n_clusters,
                        double *mean_size, int64_t *largest, uint64_t *log2_hist);

/* ---- headless view -----------------------------------------
 * The paper's program shows the run "online" through the OpenGL display of
 * the sample it adapts; a graphics API is unavailable here, so the
 * perspective view of Fig. 2, right panel, is splatted by CUDA kernels
 * into a caller buffer.  The scene is rotated by yaw about y, then pitch about x
 * (radians); the camera sits on the +z axis at eye_dist from the droplet centre and looks
 * at it; a point at view-axis distance zc projects with scale focal_px / zc onto a
 * width x height image whose principal point is the centre.  Every NP is a sphere
 * impostor of its radius, shaded 0.25 + 0.75 (n . view) times palette[type]
 * (0x00BBGGRR), nearest fragment wins; empty pixels show `droplet` inside the projected
 * disc of the droplet radius R(step) and `background` outside.  Pixels are 0xAABBGGRR
 * with AA = 0xff. */
typedef struct {
    double eye_dist, focal_px, yaw, pitch;
    int32_t width, height;               /* 1..8192 each */
    uint32_t palette[LV_MAX_TYPES];
    uint32_t background, droplet;
} lv_view;

/* zbuf_dev: DEVICE scratch of width*height*8 bytes (width*height*12 when rgba is host memory:
 * the image is staged behind the depth keys), 8-byte aligned, owned by the caller,
 * clobbered.  rgba: width*height uint32, written; host or device per on_device.
 * Synchronises when rgba is host memory; the state does not change. */
int lv_render(lv_sim *s, const lv_view *view, void *zbuf_dev, uint32_t *rgba, int on_device);

/* lv_render_surface: the LEFT panel of Fig. 2, "projection of the microdroplet surface onto
 * a plane", where "circles/ellipses (circles elongated due to the projection) correspond to
 * the NPs intersections with the microdroplet surface".  The paper does
 * not name the projection; this build takes the equirectangular map (longitude x latitude,
 * pole = z axis), which elongates circles along the longitude towards the poles as the
 * caption describes.  Pixel (px, py) of a width x height image looks at
 *   lambda = -pi + 2 pi (px + 0.5) / width,   phi = pi/2 - pi (py + 0.5) / height,
 * its direction is d = (cos phi cos lambda, cos phi sin lambda, sin phi) with the four
 * factors evaluated in fp64 and rounded once to fp32, and its surface point is
 * s = (R cl_phi c_lambda, R cl_phi s_lambda, R s_phi) -- fp32, products left to right as
 * written: R * (cos phi * cos lambda) etc. -- with R = fl32(R(step)).  NP i marks the pixel
 * iff d2 = ((sx-x)^2 + (sy-y)^2) + (sz-z)^2 < r_a * r_a (single fp32 operations, no FMA, r_a the
 * fp32 NP radius);
 * among several the smallest (bits(d2) << 32 | palette[type]) wins; a pixel no NP marks
 * shows `droplet`.  Pixels are 0xAABBGGRR with AA = 0xff.
 * scratch_dev: DEVICE scratch of width*height*8 + (width + height)*8 bytes (+ width*height*4
 * when rgba is host memory: the image is staged there), 8-byte aligned, owned by the caller,
 * clobbered.  rgba: width*height uint32, host or device per on_device.
 * Synchronises; the state does not change. */
typedef struct {
    int32_t width, height;               /* 1..8192 each */
    uint32_t palette[LV_MAX_TYPES];      /* 0x00BBGGRR per type */
    uint32_t droplet;
} lv_surface_map;

int lv_render_surface(lv_sim *s, const lv_surface_map *map, void *scratch_dev, uint32_t *rgba,
                      int on_device);

/* Batched replicas (the paper's use as a quick hypothesis tester at
 * 10^4 NPs): n_sims independent handles -- each bound to its OWN stream
 * and workspace, state loaded -- are stepped by ONE CUDA-graph launch that holds
 * steps_per_launch (1..256) steps of every replica as parallel branches.  Replicas do not
 * interact: each one's result is bit-identical to stepping it alone.  lv_batch_step(b, n)
 * enqueues n steps of all replicas on the first replica's stream (the other streams are made to
 * wait for it) and returns without synchronising; the handles stay usable for every lv_get_* /
 * lv_set_state call.  Do not call lv_step on a member while batched steps are in flight on
 * another stream.  The batch borrows the handles: destroy it before them. */
typedef struct lv_batch lv_batch;
int lv_batch_create(lv_batch **out, lv_sim **sims, int n_sims, int steps_per_launch);
int lv_batch_step(lv_batch *b, int n);
int lv_batch_destroy(lv_batch *b);

/* Status bits LV_ST_* (host uint32, written).  Synchronises. */
int lv_get_status(lv_sim *s, uint32_t *status);

/* Internal arrays for parity tests: copies min(bytes, size of the array) bytes
 * of the array `what` (LV_DBG_*) to dst (host, or device if on_device).
 * The arrays describe the last cell rebuild.  Synchronises. */
int lv_get_debug(lv_sim *s, int what, void *dst, size_t bytes, int on_device);

/* Number of kernels (own + CUB sort) one lv_step(1) enqueues; for accounting. */
int lv_launches_per_step(const lv_sim *s);

/* Measurement aid: take ONE step exactly like lv_step(1) (same kernels, direct
 * launches instead of the graph) with CUDA events between the stages on the
 * stream, synchronise, and write the device time of each stage in
 * milliseconds to ms_out (host[LV_N_STAGES]): hash (+ histogram), sort (radix
 * passes, or the histogram scan), offsets+scatter (or place + rank/gather),
 * pair force, update. */
#define LV_N_STAGES 5
int lv_step_profiled(lv_sim *s, float *ms_out);

/* Measurement aid for bench.py (CUDA events on the launching stream, inside the
 * timed region).  lv_stage_timing(s, capacity > 0): from now on every step of
 * lv_step is enqueued as direct launches of the SAME kernels (no graph) with a
 * CUDA event recorded on the stream before the first and after each of the
 * LV_N_STAGES stages; at most `capacity` steps may be taken between two reads
 * (lv_step returns LV_E_ARG beyond that).  capacity = 0 switches back to graph
 * replay and frees the events.
 * lv_read_stage_timing synchronises the stream and writes, for the steps taken
 * since the last read: ms_stage_sum (host[LV_N_STAGES]) the summed device time
 * of each stage, *ms_step_sum (host) the summed first-event-to-last-event time
 * of each step, *steps (host) their number; then resets the counter. */
int lv_stage_timing(lv_sim *s, int capacity);
int lv_read_stage_timing(lv_sim *s, double *ms_stage_sum, double *ms_step_sum, int64_t *steps);

/* Measurement aid: FP32 FMA throughput of this GPU from a register-resident
 * independent-FMA kernel on `cuda_stream`; writes TFLOP/s (host).  scratch_dev: DEVICE
 * scratch of >= 256 bytes owned by the caller.  The denominator of the pair-force kernel's
 * ALU roofline. */
int lv_measure_fp32_peak(void *cuda_stream, void *scratch_dev, double *tflops);

int lv_destroy(lv_sim *s);
const char *lv_strerror(int code);
/* Text of the last CUDA error seen by this handle (host string, library-owned). */
const char *lv_last_cuda_error(const lv_sim *s);
const char *lv_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LV_H_ */
