/* pvg.h -- C ABI of the B200-native Periodic Vibration Gaussian forward renderer.
 *
 * One hot path of arxiv 2311.18561: the time-conditioned forward splatting render
 *     I^ = Render({H_i(t)}; E, I)                 (Eq. 8; F_theta(E_o, I_o, t), L57)
 * with H(t) = {mu~(t), q, s, o~(t), c}            (Eq. 5)
 *      mu~(t) = mu + l/(2 pi) sin(2 pi (t-tau)/l) v   (Eq. 6)
 *      o~(t)  = o exp(-(t-tau)^2 / (2 beta^2))        (Eq. 7)
 * rendered by EWA projection (Eq. 2), depth sort (L70) and front-to-back
 * alpha compositing (Eq. 3) into colour, normalised depth and opacity (L87, L168).
 *
 * Every step runs in hand-written CUDA kernels for sm_100a. There is NO CPU
 * fallback: without a CUDA device every compute entry point returns PVG_ERR_CUDA.
 * All functions return 0 (PVG_OK) or a negative pvg_status; nothing throws or
 * aborts across this boundary. One render at a time per scene; distinct scenes
 * are independent. Readings of the points the paper leaves open are in DESIGN.md.
 */
#ifndef PVG_H_
#define PVG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum pvg_status {
  PVG_OK = 0,
  PVG_ERR_NULL = -1,              /* a required pointer is NULL */
  PVG_ERR_BAD_DESC = -2,          /* n == 0 or n >= 2^31, cycle <= 0 or NaN, sh_degree outside 0..3 */
  PVG_ERR_BAD_CAMERA = -3,        /* non-positive or non-finite size / focal length, size > 32768 */
  PVG_ERR_OOM = -4,               /* device allocation failed */
  PVG_ERR_INSTANCE_OVERFLOW = -5, /* tile instances M >= 2^32 */
  PVG_ERR_CUDA = -6,              /* CUDA runtime error (or no device); see pvg_last_cuda_error */
  PVG_ERR_BAD_OPTION = -7,
  PVG_ERR_BAD_STATE = -8,         /* non-finite t or dt, rho_min < 0, rho_max < rho_min, unknown target */
  PVG_ERR_TOO_LARGE = -9          /* pvg_sort_pairs_static: more pairs than the static scratch holds; see pvg_last_cuda_error */
} pvg_status;

typedef struct pvg_scene pvg_scene; /* opaque; owns device copies of the model and a growable workspace */

/* The model theta = per-point {mu, q, s, o, c, tau, beta, v} + cycle length l
 * (PAPER.md:L110). All arrays are dense, row-major float32, read once by
 * pvg_create_scene (the caller may free them on return). */
typedef struct pvg_scene_desc {
  uint64_t n;           /* points, 1 .. 2^31-1 */
  const float *mu;      /* [n][3]  world position mu  */
  const float *quat;    /* [n][4]  rotation (w,x,y,z); normalised by the library (L79)      */
  const float *scale;   /* [n][3]  std-devs s > 0, already activated        (L79)           */
  const float *opacity; /* [n]     o in [0,1], already activated            (L61)           */
  const float *sh;      /* [n][16][3] degree-3 real SH, coefficient-major, channel-minor    */
  const float *tau;     /* [n]     life peak tau                            (L95)           */
  const float *beta;    /* [n]     lifespan beta > 0; +INF = never fades    (L110, L114)    */
  const float *vel;     /* [n][3]  v = d mu~/dt at tau                      (L110)          */
  float cycle;          /* l > 0; +INF selects the linear model mu + (t-tau) v (L336)       */
  int sh_degree;        /* 0..3: bands above it are ignored */
  int pointers_on_device; /* 0: host pointers, 1: device pointers (copied either way) */
} pvg_scene_desc;

/* Camera pose [E_o, I_o]. Pinhole, no distortion.
 * p_cam = R p_world + T with world_to_cam = row-major 3x4 [R|T]; +z forward,
 * +x right, +y down. Pixel (i,j) has its centre at (i+0.5, j+0.5). */
typedef struct pvg_camera {
  int width, height;      /* 1 .. 32768 */
  float fx, fy, cx, cy;   /* pixels */
  float world_to_cam[12];
  float znear;            /* cull p_cam.z <= znear; <= 0 selects the default 0.2 */
  float bg[3];            /* constant background colour: rgb = C + (1 - O) bg (L168 with constant f_sky) */
} pvg_camera;

/* ---- plumbing: device memory and stream come from the caller (PyTorch) -------------------- */

/* Device allocator hooks (process-wide; set before the first pvg_create_scene).
 * alloc returns a device pointer aligned to >= 256 B or NULL; `stream` is the
 * cudaStream_t the memory will first be used on. NULL hooks restore cudaMalloc/cudaFree. */
typedef void *(*pvg_alloc_fn)(size_t bytes, void *stream, void *user);
typedef void (*pvg_free_fn)(void *ptr, void *user);
int pvg_set_allocator(pvg_alloc_fn alloc_fn, pvg_free_fn free_fn, void *user);

/* cudaStream_t (as void*) that pvg_render enqueues on; default: the legacy default stream. */
int pvg_set_stream(pvg_scene *scene, void *cuda_stream);

/* ---- the path ---------------------------------------------------------------------------- */

/* Copies the model to the device and re-lays it out (structure of arrays, float4). */
int pvg_create_scene(const pvg_scene_desc *desc, pvg_scene **out);

/* Renders the frame at timestamp t. Outputs are caller-owned DEVICE buffers:
 *   out_rgb [3][H][W], out_depth [H][W] (sum T a z / sum T a, 0 where alpha == 0), out_alpha [H][W] (O = sum T a).
 * Any of the three may be NULL (not written). Work is enqueued on the scene's stream; the call
 * blocks once, to read the instance count M back (it sizes the sort buffers), and returns with
 * the blend kernel still in flight. */
int pvg_render(pvg_scene *scene, const pvg_camera *cam, float t, float *out_rgb, float *out_depth,
               float *out_alpha);

/* Which state of the model is rendered:
 *   dt == 0: H(t) = { mu~(t), q, s, o~(t), c } (Eq. 5-7) -- what pvg_render draws.
 *   dt != 0: the temporal-smoothing estimate of the state at t from the state at t1 = t - dt,
 *            H^(t) = { mu~(t1) + vbar dt, q, s, o~(t1), c } (Eq. 12), with the average velocity
 *            vbar = v exp(-rho / 2) (Eq. 10) and the staticness rho = beta / l (L112).
 *   rho_min, rho_max: only points with rho_min <= rho <= rho_max are drawn; {0, +INF} draws all. The paper
 *            removes rho < 1 to keep the static part of a scene (L192) and thresholds rho to tell dynamic
 *            points (L118). beta = +INF counts as rho = +INF; cycle = +INF with finite beta as rho = 0. */
typedef enum pvg_target {
  PVG_TARGET_COLOR = 0,   /* out_rgb = C + (1 - O) background, out_depth = sum T a z / sum T a */
  /* SURVEY 8(f-2), "flexible rendering ... by replacing the color c in Eq. (3)" with the
   * quantities of the paper's dynamic element analysis (L298): out_rgb = sum T a vbar_cam, the average velocity
   * vbar = v exp(-rho/2) (Eq. 10) rotated into camera axes (x right, y down, z forward; its x, y components are
   * the projection onto the plane parallel to the camera plane that the paper colour-codes); out_depth =
   * sum T a clamp(rho, 0, 2), the staticness map. Plain sums of Eq. 3: no background, no normalisation;
   * out_alpha = O as always. The record's colour slot holds vbar_cam in this mode. */
  PVG_TARGET_DYNAMICS = 1
} pvg_target;
typedef struct pvg_state {
  float t, dt, rho_min, rho_max;
  int target; /* pvg_target */
} pvg_state;
int pvg_render_state(pvg_scene *scene, const pvg_camera *cam, const pvg_state *state, float *out_rgb,
                     float *out_depth, float *out_alpha);

/* Sky: "a high-resolution learnable environment cube map f_sky(d) = c_sky as the background.
 * The final color is C_f = C + (1 - O) f_sky(d)". cube = [6][res][res][3] floats (host or
 * device; copied), NULL switches the sky off (the camera's constant bg is used again). d is the pixel-centre
 * ray in WORLD coordinates, R^T ((x - cx)/fx, (y - cy)/fy, 1). Layout (the paper fixes none): face =
 * 2 a + (d_a < 0) for the axis a of largest |d_a| (faces +x, -x, +y, -y, +z, -z; ties: lowest axis);
 * u = d_b / |d_a|, v = d_c / |d_a| with (b, c) the next two axes in cyclic order; texel (i, j) = cube[face][j][i]
 * has its centre at u = (2 i + 1)/res - 1, v = (2 j + 1)/res - 1; bilinear between the four nearest centres,
 * clamped to the face (no filtering across faces). Synchronises the scene's stream. */
int pvg_set_sky(pvg_scene *scene, const float *cube, int res, int on_device);

/* Same frame into HOST buffers (pinned or pageable): renders into library-owned device images,
 * copies them back and synchronises the stream before returning. */
int pvg_render_host(pvg_scene *scene, const pvg_camera *cam, float t, float *host_rgb,
                    float *host_depth, float *host_alpha);

/* Pipelined variant for frame streams: enqueues the render and the device-to-host copies (on an
 * internal copy stream, from one of two library-owned device images) and returns without waiting,
 * so the copy of frame k overlaps the render of frame k + 1. The host buffers should be pinned
 * (pageable memory makes the copies synchronous) and must not be read before pvg_wait_host, which
 * blocks until every pending copy of the scene has landed. At most two frames are in flight: the
 * third call reuses the first one's device image after its copy has left. */
int pvg_render_host_async(pvg_scene *scene, const pvg_camera *cam, float t, float *host_rgb,
                          float *host_depth, float *host_alpha);
int pvg_wait_host(pvg_scene *scene);

/* Frames in flight. Frames (camera, t) are independent, but one scene renders them one
 * after another: its workspace holds one frame and the host waits once per frame for the frame's sizes. A FORK
 * is a second scene handle on the SAME model (the re-laid-out Gaussians are shared and reference-counted: no
 * copy, no extra model memory) with its own workspace, side streams and options (copied from the parent at the
 * fork; the sky cube map is not inherited). Rendering alternate frames through a scene and its fork, each on
 * its own stream (pvg_set_stream), keeps two frames in flight: the latency-bound kernels of one overlap the
 * bandwidth- and issue-bound kernels of the other (config 3: +8% frames/s with two, nothing more with three).
 * Each handle is destroyed with pvg_destroy, in any order; the model goes with the last one. A handle is not
 * thread-safe; different handles may be used from different threads. Results are those of pvg_render. */
int pvg_fork_scene(pvg_scene *scene, pvg_scene **out);

int pvg_destroy(pvg_scene *scene);

/* ---- options ------------------------------------------------------------------------------ */
typedef enum pvg_option {
  /* 1 (default): sort the Gaussians by depth first (n keys, 32 bits), emit tile instances in that
   *    order, then radix-sort the M instances on the tile-id bits only.
   * 0: emit in index order and radix-sort all 32 + ceil(log2 tiles) key bits of the M instances.
   * Both are the same stable LSD sort and give bit-identical sorted lists and ranges. */
  PVG_OPT_PRESORT_DEPTH = 1,
  /* 1: keep a copy of the unsorted (key,value) list for pvg_debug_view (default 0). */
  PVG_OPT_KEEP_UNSORTED = 2,
  /* 0 (default): no events. 1: record CUDA events around every kernel of the last render
   * (pvg_kernel_times_ms, pvg_stage_times_ms; without it they report nothing). 2: keep the records of
   * EVERY render until pvg_kernel_times_ms reads (and clears) them. A measurement hook: the records cost
   * ~4% of a 1 ms frame, and far more (measured +34%) in the pvg_render_host_async pipeline, where they
   * interleave with the image copies. */
  PVG_OPT_KERNEL_EVENTS = 3,
  /* 1: the blend also counts its (pixel, list entry) evaluations (pvg_blend_counters); measurement
   *    only -- the counting variant is a separate kernel instantiation (default 0). */
  PVG_OPT_COUNT_PAIRS = 4,
  /* 1 (default): with PRESORT_DEPTH=1 and at most 65536 tiles, an instance travels through the
   *    tile-id passes as (u16 tile id, u32 Gaussian index) instead of the 64-bit key + index: its
   *    depth bits are already in order and would be dead payload. pvg_debug_view rebuilds the
   *    64-bit keys on demand. 0: always carry the 64-bit keys. Results are identical. */
  PVG_OPT_COMPACT_KEYS = 5,
  /* 1 (default): with PRESORT_DEPTH=1 and at most 256 blocks of 8x8 tiles (images up to 2048x2048
   *    pixels or the same area), the per-tile lists are built from one entry per (Gaussian, block)
   *    -- block id, Gaussian index, 64-bit mask of the covered tiles -- instead of one key per
   *    (Gaussian, tile): the entries are split by block with one onesweep digit pass and expanded
   *    into the tile lists by ballots, in depth order. The sorted list and the ranges are
   *    bit-identical to those of the 64-bit key sort; the unsorted key list and the per-instance
   *    offsets are not intermediates of this mode (pvg_debug_view produces them on demand).
   * 0: one key per (Gaussian, tile) as above. */
  PVG_OPT_BLOCK_BINS = 6,
  /* 1 (default): while it stages a batch of its list, the blend drops the entries whose ellipse
   *    { alpha >= 1/255 } cannot reach any pixel centre of the tile (the lists are built from axis-aligned
   *    rectangles; a quarter to a half of the entries a tile consumes only cover it with their rectangle).
   *    Such an entry is rejected at every pixel anyway, so the images are bit-identical; the test is
   *    conservative by a rounding margin. 0: every listed entry is evaluated at every pixel. */
  PVG_OPT_BLEND_CULL = 7,
  /* k >= 1 (default 1): with KERNEL_EVENTS on, record the launches of every k-th render only, counted from the
   *    call that sets this option or KERNEL_EVENTS (renders 0, k, 2k, ...). An event record between two kernels
   *    costs about 2 us of stream time -- 3.6% of a 1 ms frame with ~16 records -- so a long timed loop samples. */
  PVG_OPT_EVENT_STRIDE = 8,
  /* The band of tile rows [BEGIN, END) a render covers (the within-frame multi-GPU split --
   *    every GPU holds the scene, preprocesses all N Gaussians but duplicates only into the tiles of its own band,
   *    and writes only the pixel rows [16*BEGIN, min(16*END, H)) of the output images; the other rows are left
   *    untouched, so bands rendered one after another into the same images add up to the full frame bit for bit).
   *    Defaults 0 and 0; END = 0 (or beyond the image) means "to the last tile row". A band that is empty for the
   *    camera of a render (BEGIN >= its tile rows) makes that render return PVG_ERR_BAD_STATE.
   *    In a band render the per-Gaussian counts, M and the ranges describe the band's tiles only. */
  PVG_OPT_TILE_ROW_BEGIN = 9,
  PVG_OPT_TILE_ROW_END = 10,
  /* k > 0 (default 2), BLOCK_BINS mode: lazy tile lists. Front-to-back compositing stops a pixel at T < 1e-4, so a
   *    tile reads its depth-sorted list only as far as its last live pixel needs -- at config 3 a few hundred of
   *    its ~30 000 entries. The lists are therefore first written only as far as the first k chunks (512 block
   *    entries each, in depth order) of every 8x8-tile block reach; the blend runs on these prefixes; the tiles
   *    that still have a live pixel at the end of their prefix park their per-pixel state, get the REST of their
   *    lists written (only those tiles), and resume. Every pixel sees the same entries in the same order with the
   *    same arithmetic: the images are bit-identical to k = 0, and every list position that is written holds what
   *    the complete list holds there. pvg_debug_view writes the remainder on demand, so vals_sorted is always
   *    every tile's whole list. 0: write the complete lists before the blend. */
  PVG_OPT_LAZY_CHUNKS = 11,
  /* d >= 1 (default 16), with LAZY_CHUNKS > 0: lazy emission. Only the first 1/d of the block entries, in depth order
   *    (whole tiles of 4096; at least twice what the first LAZY_CHUNKS chunks of every block hold, so that small scenes
   *    do not park for want of entries), is formed and split by block before the first blend phase; a block's chunk counts for
   *    that phase only if all of its 512 entries exist. The entries behind the slab are formed only if a tile was
   *    parked (the launch checks the count on the device). 1: form all entries up front. */
  PVG_OPT_LAZY_SLAB = 12,
  /* 1 (default 0), BLOCK_BINS mode: exact tile lists. A Gaussian's tile rectangle is the bounding box
   *    of the region where its alpha can reach 1/255; towards the corners it holds tiles the region does not touch
   *    (a quarter of all instances at config 3, half at config 4). With this option a Gaussian is listed only in the
   *    tiles whose box of pixel centres the region can reach: every block entry's tile mask is refined by an fp32 test
   *    taken with individually rounded operations (the oracle takes the same ones), the per-tile counts are counted
   *    from the refined masks and the ranges rebuilt from them. A dropped (Gaussian, tile) pair contributes to no
   *    pixel, so the images are bit-identical; counts, M, the sorted list and the ranges are those of the exact lists
   *    (pvg_debug_view; no unsorted list in this mode). Implies complete lists and eager records (LAZY_CHUNKS is
   *    ignored): with lazy lists the same test already runs inside the blend on the few entries a tile consumes
   *    (BLEND_CULL), which is cheaper by two orders of magnitude -- this mode is for consumers of the lists themselves. */
  PVG_OPT_EXACT_TILES = 13,
  /* 0, 1 (default: on for scenes of at least 2^19 Gaussians, where it pays) or 2 (always on), with LAZY_CHUNKS > 0:
   *    front-first depth order. The first blend phase consumes the first slab of the
   *    block entries in depth order, and those belong to the few Gaussians nearest the camera (about 1 % of the
   *    survivors at config 3: near Gaussians are large on screen). So the frame orders, scans and bins only that front:
   *    preprocess's last CTA picks a depth-key threshold from a histogram of the entries over the top key bits such
   *    that the Gaussians below it own more than the slab; the pairs below the threshold are compacted in index
   *    order (the sort stays stable) and radix-sorted. The pairs at and beyond the threshold are compacted, sorted
   *    behind the front and scanned only if a tile was parked (or pvg_debug_view asks): a sorted front followed by a
   *    sorted back is the sorted whole, the threshold being a key value, so the visiting order, the offsets, the
   *    lists and the images are bit-identical to 0. 0: sort all survivors up front. */
  PVG_OPT_LAZY_DEPTH = 14
} pvg_option;
int pvg_set_option(pvg_scene *scene, int option, int64_t value);

/* ---- test and measurement hooks (not part of the paper's problem) ------------------------- */

/* Device views of the last render's intermediates, valid until the next call on the scene.
 * With COMPACT_KEYS in effect this call launches two small kernels that rebuild the 64-bit key
 * lists and synchronises the stream: a debugging call, not for timed loops (pvg_frame_stats). */
typedef struct pvg_debug {
  uint64_t n;                    /* points */
  uint64_t num_instances;        /* M = sum of counts */
  uint32_t tiles_x, tiles_y;     /* ceil(W/16), ceil(H/16) */
  uint32_t sort_begin_bit, sort_end_bit; /* key bits the M-instance sort covered */
  const float *record;           /* [n][12] (mx,my,z,o~ | a,b,c,hx | r,g,b,hy); all 0 if culled */
  const uint32_t *counts;        /* [n] tiles touched (0 if culled) */
  const uint32_t *visit_order;   /* [n] Gaussian index visited at position r; NULL = identity (PRESORT_DEPTH=0) */
  const uint32_t *offsets;       /* [n] exclusive instance offset of visit position r */
  const uint64_t *keys_unsorted; /* [M] (tile << 32 | fp32 bits of z), NULL unless KEEP_UNSORTED */
  const uint32_t *vals_unsorted; /* [M] Gaussian index */
  const uint64_t *keys_sorted;   /* [M] */
  const uint32_t *vals_sorted;   /* [M] */
  const uint32_t *ranges;        /* [tiles][2] = [begin, end) of each tile in the sorted list */
} pvg_debug;
int pvg_debug_view(pvg_scene *scene, pvg_debug *out);

/* Stages of the last render; ms[] from CUDA events on the scene's stream (synchronises). */
enum {
  PVG_STAGE_PREPROCESS = 0, /* a1 */
  PVG_STAGE_DEPTH_SORT = 1, /* a3, the n-key part (PRESORT_DEPTH=1) */
  PVG_STAGE_DUPLICATE = 2,  /* a2 scan + key emission */
  PVG_STAGE_SORT = 3,       /* a3, the M-instance part */
  PVG_STAGE_RANGES = 4,     /* a4 */
  PVG_STAGE_BLEND = 5,      /* a5 */
  PVG_NUM_STAGES = 6
};
int pvg_stage_times_ms(pvg_scene *scene, float ms[PVG_NUM_STAGES]);

/* Per-kernel device times of the last render, in launch order. Fills up to `cap` entries of
 * names (static strings), stage ids and milliseconds; returns the number of launches (>= 0)
 * or a negative pvg_status. */
int pvg_kernel_times_ms(pvg_scene *scene, int cap, const char **names, int *stages, float *ms);

/* The same launches as a timeline: start (relative to the first launch of the frame) and duration of each, in
 * launch order, so that gaps and the overlap of the side stream are visible. Same return convention. */
int pvg_kernel_timeline_ms(pvg_scene *scene, int cap, const char **names, float *start_ms, float *dur_ms);

/* Sizes of the last render, no device work: out = {points n, tile instances M (of the rectangles), tiles_x, tiles_y,
 * block entries (BLOCK_BINS mode, else 0), list mode: 0 = 64-bit keys, 1 = compact keys, 2 = block entries, 3 = block
 * entries with exact tile lists, surviving Gaussians S (PRESORT_DEPTH=1, else 0), tiles the first blend phase of the
 * lazy lists parked (LAZY_CHUNKS; valid once the frame has completed on the stream), instances of the exact lists
 * (EXACT_TILES; valid once the frame has completed), pairs the front-first depth order sorted up front (LAZY_DEPTH,
 * else 0)}. */
int pvg_frame_stats(pvg_scene *scene, uint64_t out[10]);

/* Work done by the last blend when PVG_OPT_COUNT_PAIRS=1: out[0] = (pixel, list entry) pairs
 * evaluated before the pixel stopped, out[1] = pairs that contributed (alpha >= 1/255). */
int pvg_blend_counters(pvg_scene *scene, uint64_t out[2]);

/* The onesweep LSD radix sort as a primitive: stable sort of n (key,value) pairs on key bits
 * [begin_bit, end_bit). All pointers are DEVICE buffers of n elements; the sorted result is
 * written to keys_out/vals_out, keys_in/vals_in are clobbered. Runs on `cuda_stream` and
 * synchronises it. */
int pvg_sort_pairs(uint64_t n, uint64_t *keys_in, uint32_t *vals_in, uint64_t *keys_out,
                   uint32_t *vals_out, int begin_bit, int end_bit, void *cuda_stream);

/* The same sort for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): its scratch -- digit histograms, tickets, look-back words -- lives in a file-scope device array
 * of the library, 4.01 MB that every GPU which loads the library holds until the process exits, enough for
 * n <= PVG_SORT_STATIC_MAX_N pairs and any bit range. Calls no cudaMalloc, cudaFree or allocating library routine.
 *   - Same arguments, layouts and result as pvg_sort_pairs (DEVICE buffers of n elements owned by the caller; the
 *     sorted pairs land in keys_out / vals_out, keys_in / vals_in are clobbered), on the current device.
 *   - n > PVG_SORT_STATIC_MAX_N: returns PVG_ERR_TOO_LARGE, nothing is enqueued, pvg_last_cuda_error() says why.
 *   - ASYNCHRONOUS: the work is enqueued on `cuda_stream` and the call returns; it does not synchronise (unlike
 *     pvg_sort_pairs). Errors of the kernels themselves surface at the caller's next synchronisation.
 *   - Every call on a device shares the one array (it keeps the last call's contents; the call clears what must
 *     start at zero, on the stream): two calls that overlap on the GPU -- different streams without an ordering
 *     between them, or different host threads -- RACE on it. Calls on one stream are ordered and safe. */
#define PVG_SORT_STATIC_MAX_N (1u << 20)
int pvg_sort_pairs_static(uint64_t n, uint64_t *keys_in, uint32_t *vals_in, uint64_t *keys_out,
                          uint32_t *vals_out, int begin_bit, int end_bit, void *cuda_stream);
uint64_t pvg_sort_pairs_static_max_n(void);   /* PVG_SORT_STATIC_MAX_N as the library was built */

/* Measurement hook for the roofline of the ALU-bound blend ("calibrate with an FFMA microbenchmark on
 * the box"): runs a register-only kernel on the current device (8 CTAs of 256 threads per SM, 8 independent chains
 * per thread, a few ms) and reports the best of four timed launches as thread-level instructions per second.
 *   mode 0: FFMA only (three register operands);  mode 1: FFMA and LOP3 alternating (FMA pipe + ALU pipe: the issue
 *   rate an instruction mix like the blend's can reach);  mode 2: packed FFMA2 (fma.rn.f32x2; one instruction = two FMAs,
 *   counted once). sm_count (may be NULL) receives cudaDevAttrMultiProcessorCount. Synchronises `cuda_stream`. */
int pvg_calibrate_fp32(int mode, void *cuda_stream, double *thread_instr_per_s, int *sm_count);

/* Test hook: guard bands. After pvg_guard_bands(1) every device allocation the library makes (model, workspace) carries
 * 4096 bytes of a known pattern in front and behind; pvg_check_guards synchronises the device and reports how many live
 * allocations have a damaged band (a kernel wrote out of bounds) and how many were checked. A stand-in for
 * compute-sanitizer's memcheck where that tool is not available; off by default, process-wide. */
int pvg_guard_bands(int enable);
int pvg_check_guards(uint64_t *damaged_allocations, uint64_t *checked_allocations);

/* Debug helper so that bindings need no CUDA runtime of their own: synchronous copy of `bytes`
 * from a device pointer (e.g. a pvg_debug view) into host memory. */
int pvg_memcpy_d2h(void *host_dst, const void *device_src, size_t bytes);

const char *pvg_strerror(int code);
const char *pvg_last_cuda_error(void); /* text of the last CUDA error seen by this thread's calls */
int pvg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PVG_H_ */
