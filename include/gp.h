/* gp.h — C ABI of the B200-native batched per-agent perspective renderer ("Gigapixel" hot path).
 *
 * What the library computes: O_pixel(S_t, i) of PAPER.md:60-62 (§3.1) — the simulator state
 * S_t = (A_t, M, L_t) rendered into the ego-centric perspective view of every agent i of every
 * parallel world, "thousands of environments ... in a single batched launch",
 * cuboids for agents, planar strips for road segments, one directional light, per-instance
 * attributes, images "exposed directly as a batched GPU tensor ... no per-step
 * CPU transfer" with configurable resolution and camera.  The per-pixel arithmetic
 * is the written contract C0-C8 of DESIGN.md §3 (the paper gives no formula).
 *
 * Conventions
 *  - Every function returns an int status: GP_OK (0) or a negative GP_ERR_* code.  Argument errors
 *    write nothing.  gp_error_string(code) returns a static string; after GP_ERR_CUDA it contains
 *    the CUDA error text of the calling thread's last failure.
 *  - "DEVICE" pointers are CUDA device pointers on the context's device; "HOST" pointers are plain
 *    host memory.  The library never frees or keeps caller memory.  Output buffers are caller-owned.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls enqueue
 *    work on it and return without synchronising, except where stated.
 *  - Only sm_100 (B200) devices are accepted; there is no fallback path of any kind.
 *  - Views are ordered world-major, then agent, then camera of the rig (gp_camera_rig_set; one front
 *    camera by default): view = (world * agents_per_world + agent) * n_cams + cam.
 */
#ifndef GP_H_
#define GP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    GP_OK = 0,
    GP_ERR_ARG = -1,        /* NULL / non-positive / inconsistent argument                   */
    GP_ERR_ALIGN = -2,      /* an output or input pointer is not 16-byte aligned             */
    GP_ERR_STATE = -3,      /* call order: render / update before gp_scene_upload            */
    GP_ERR_RANGE = -4,      /* world range outside the scene, agents != agents_per_world     */
    GP_ERR_CUDA = -5,       /* a CUDA runtime call failed (text via gp_error_string)         */
    GP_ERR_ARCH = -6,       /* the device is not compute capability 10.x                     */
    GP_ERR_NOMEM = -7,      /* device or host allocation failed                              */
    GP_ERR_LIMIT = -8       /* gp_render_static: scene or image larger than its fixed scratch */
};

/* gp_set_option keys */
enum {
    GP_OPT_PATH = 1,        /* GP_PATH_FAST (default) or GP_PATH_BRUTE                        */
    GP_OPT_STATS = 2,       /* 1: count executed ray/primitive tests and listed pairs         */
    GP_OPT_TIMING = 3,      /* n > 0: bracket every n-th launch of each kernel with CUDA events
                               (gp_kernel_time); 0: off                                         */
    GP_OPT_STAGE_CAP = 4,   /* list entries per view staged in shared memory (>= 1); longer lists read their tail from
                               global memory.  0 = automatic, never more than the primitives per world.  Ray variant:
                               48 for images of up to 1024 pixels (32 x 32), 64 up to 64 x 64, else 128 - except that a
                               crowded world (>= 400 primitives, gather mode, 4-warp CTAs) gives up staged entries, down
                               to 80, when that lets 8 CTAs share an SM instead of 7.  Raster variant: always 128 */
    GP_OPT_STRIP_PX = 5,    /* target pixels per warp strip of the render pass; 0 = automatic   */
    GP_OPT_GATHER = 6,      /* how a strip works off its list: 1 gather the overlapping entries first, one lane
                               per (flat quad, row); 0 entry by entry; -1 (default) chosen from the image size
                               and the primitives per world                                        */
    GP_OPT_VARIANT = 8,     /* render pass: GP_VARIANT_RAY (pixel-major strips), GP_VARIANT_RASTER (primitive-major
                               tiles with a depth buffer, PAPER.md:62 / :319) or -1 (default) = the ray variant for
                               every shape: the raster variant measured 7-41 % slower on all six shapes tried
                               (profiles/r02_raster_vs_ray.md) and is kept as the selectable alternative.
                               Results are bit-identical.                                            */
    GP_OPT_TILE_PX = 9,     /* raster variant: target pixels per tile; 0 = automatic                   */
    GP_OPT_PIPELINE = 10,   /* n >= 1 world chunks per gp_render_batch; with n > 1 the culls of chunks 1.. run on a
                               library-owned high-priority stream concurrently with the renders of earlier chunks.
                               Default 1 (serial): the overlap measured slower on every workload */
    GP_OPT_LIST_CAP = 11,   /* n > 0: the per-view lists of the cull hold at most min(n, primitives per world) entries, so the
                               library-owned scratch is views x n x 64 B instead of views x P x 64 B (worlds with thousands of
                               static segments of which a view sees few).  A view whose list does not fit is rendered by the
                               brute-force kernel in a repair pass after the render pass: results are unchanged, that view is
                               slow.  0 (default): n = P, no repair pass.  Set before gp_reserve / the first render */
    GP_OPT_SPHERES = 7      /* are records with shape == GP_SHAPE_SPHERE drawn?  -1 (default) automatic: yes iff the
                               uploaded scene held a sphere or gp_statics_update has run since the upload (its
                               records are device memory the host never inspects); 1 yes; 0 no: sphere records
                               are skipped by every path alike (the render pass then runs without the sphere
                               branch, which costs the box-only case a few per cent)                 */
};
enum {                      /* kernel ids of gp_kernel_time                                   */
    GP_KERNEL_UPDATE = 0,   /* a0 pose update + shading table                                 */
    GP_KERNEL_CULL = 1,     /* a1 camera setup + a2 frustum cull and compaction               */
    GP_KERNEL_RENDER = 2,   /* a3-a9 render pass (fast path)                                  */
    GP_KERNEL_BRUTE = 3,    /* brute-force kernel                                             */
    GP_KERNEL_DYNAMICS = 4, /* gp_dynamics_step                                               */
    GP_KERNEL_OBSERVE = 5   /* gp_observe_vec                                                 */
};
enum { GP_VARIANT_RAY = 0, GP_VARIANT_RASTER = 1 };
enum {
    GP_PATH_FAST = 0,       /* cull + compaction, list staged in shared memory, strip render  */
    GP_PATH_BRUTE = 1       /* one thread per pixel, every primitive of the world, no culling */
};

typedef struct gp_ctx gp_ctx;   /* opaque, library-owned */

/* Scene-wide constants (C1, C2, C4, C8).  Plain data, copied at upload. */
typedef struct {
    int32_t n_worlds;           /* Wn >= 1                                                    */
    int32_t agents_per_world;   /* A >= 1: primitives 0..A-1 of a world are the agents        */
    int32_t quads_per_world;    /* Q >= 0: primitives A..A+Q-1 are static                     */
    float cam_height;           /* camera z, metres (1.6)                                     */
    float t_max;                /* far plane on planar depth, metres (100); +inf allowed      */
    float light[3];             /* unit vector towards the light (0.48, 0.36, 0.8)            */
    float ambient;              /* in [0,1] (0.25)                                            */
    uint8_t palette[8][3];      /* RGB of class 0 sky, 1 ground, 2 marking, 3 vehicle, 4-7 user
                                   classes (pedestrian, cyclist, obstacle, light: PAPER.md:62)  */
} gp_scene_desc;

#define GP_MAX_CAMS 8

/* One camera of the per-agent rig (C2; PAPER.md:317 "the ego camera is an entity", :319
 * "number of cameras configurable", :434 front / front-left / front-right / rear).  16 bytes. */
typedef struct {
    float cos_yaw_off, sin_yaw_off;   /* yaw offset from the agent's heading, positive = to the left   */
    float mount;                      /* position on the agent's x axis in half lengths: +1 front-centre,
                                         0 centre, -1 rear-centre                                      */
    float pad;
} gp_camera;

enum { GP_SHAPE_BOX = 0, GP_SHAPE_SPHERE = 1 };

/* One primitive (C1; "vehicles and static objects use cuboids, road segments use
 * planes, and traffic lights use spheres").  GP_SHAPE_BOX: an oriented box; hz == 0 makes it a flat quad.
 * GP_SHAPE_SPHERE: a sphere of radius hx about the centre (hy, hz and the heading are ignored), drawn
 * unshaded in its class colour (lights are emissive, C8).  48 bytes. */
typedef struct {
    float cx, cy, cz;           /* centre, world frame: z up                                  */
    float hx, hy, hz;           /* half extents along the box axes, >= 0                      */
    float cos_yaw, sin_yaw;     /* heading of the box x axis                                  */
    int32_t cls;                /* class id written to the class plane (0..7)                 */
    int32_t inst;               /* instance id written to the instance plane                  */
    int32_t shape;              /* GP_SHAPE_BOX or GP_SHAPE_SPHERE                            */
    int32_t pad;
} gp_prim;

/* Create a context on CUDA device `cuda_device`.  GP_ERR_ARCH unless it is sm_100. */
int gp_create(gp_ctx **out, int cuda_device);

/* Free every device allocation of the context.  Synchronises the device. */
int gp_destroy(gp_ctx *ctx);

int gp_set_option(gp_ctx *ctx, int key, int value);

/* Step a0 (scene residency).  Copies desc, h_agents [Wn][A] and h_quads [Wn][Q] (HOST; h_quads may be
 * NULL iff Q == 0) into library-owned device memory as one table [Wn][A+Q], derives the per-primitive
 * shading table (C8) on the device and resets every camera pitch to 0.  The host arrays are copied
 * into a library-owned staging buffer before the call returns, so they may be freed at once.
 * (Re)allocates device memory: not for use inside a timed loop. */
int gp_scene_upload(gp_ctx *ctx, const gp_scene_desc *desc, const gp_prim *h_agents,
                    const gp_prim *h_quads, void *stream);

/* Step a0 (pose update).  d_pose: DEVICE [Wn][A][4] fp32 = (cx, cy, cos yaw, sin yaw) of every agent;
 * overwrites those four fields of the agent records and refreshes their shading table.  16-byte
 * aligned.  No host transfer. */
int gp_agents_update(gp_ctx *ctx, const float *d_pose, void *stream);

/* Replace static primitives from device memory.  d_prims: DEVICE [Wn][n] gp_prim records (16-byte aligned) that
 * overwrite static slots [q_begin, q_begin + n) of every world (primitives A + q_begin ...), verbatim; their
 * shading tables are refreshed.  Fields are NOT validated (cls is masked to 0..7; a shape other than
 * GP_SHAPE_SPHERE is a box).  Spheres introduced here are drawn: after this call the render pass runs with its
 * sphere branch (see GP_OPT_SPHERES to declare that no sphere will ever be written).  With agents_per_world = 1
 * this gives the paper's one-world-per-ego layout: the ego is the agent, everything else static
 * slots refreshed per step without a host transfer. */
int gp_statics_update(gp_ctx *ctx, const gp_prim *d_prims, int n, int q_begin, void *stream);

/* Static map from polylines, on the device (C1p; "lane polylines ... thin planar strips",
 * :331 "road geometry, encoded as polyline segments").  d_points: DEVICE [Wn][n_lines][pts_per_line][2] fp32
 * (x, y), 8-byte aligned.  Segment s of line l of world w overwrites static primitive number
 * q = q_begin + l * (pts_per_line - 1) + s of that world (primitive A + q): a flat quad centred on the segment's
 * midpoint, half length along the segment, heading = the normalised segment direction ((1, 0) for a zero-length
 * segment), half width `half_width`, height `z`, class `cls`, instance A + q; its shading table is refreshed.
 * q_begin >= 0 and q_begin + n_lines * (pts_per_line - 1) <= quads_per_world, pts_per_line >= 2.  No host
 * transfer: a new map can be installed per episode without leaving the device. */
int gp_statics_from_polylines(gp_ctx *ctx, const float *d_points, int n_lines, int pts_per_line,
                              float half_width, float z, int cls, int q_begin, void *stream);

/* Camera pitch per view.  d_pitch_cs: DEVICE [Wn][A][2] fp32 = (cos p, sin p), positive = nose up;
 * NULL resets every camera to pitch 0.  Copied on `stream`. */
int gp_cameras_set(gp_ctx *ctx, const float *d_pitch_cs, void *stream);

/* The camera rig shared by all agents: h_rig HOST [n_cams], 1 <= n_cams <= GP_MAX_CAMS, copied before
 * the call returns.  Default after gp_create: one camera (1, 0, +1) = front-centre, looking ahead.
 * Takes effect for renders enqueued afterwards; the pitch set by gp_cameras_set applies to every
 * camera of an agent. */
int gp_camera_rig_set(gp_ctx *ctx, int n_cams, const gp_camera *h_rig);

/* Steps a1-a9.  Renders the views of worlds [world_begin, world_begin + n_worlds) at H x W pixels with
 * horizontal field of view fov_rad (vertical follows from square pixels).  `agents` must equal
 * agents_per_world.  Outputs (DEVICE, 16-byte aligned, n = n_worlds*agents*n_cams views, row-major,
 * row 0 = top):
 *   d_class    [n][H][W]    uint8   0 sky, 1 ground, else the winning primitive's cls
 *   d_instance [n][H][W]    int32   the winning primitive's inst; -1 for ground and sky
 *   d_depth    [n][H][W]    float   planar depth of the nearest hit; 0 for sky
 *   d_rgb      [n][3][H][W] uint8   shaded colour, planar; NULL skips the plane
 * 1 <= H, W <= 4096.  The fast path needs W >= 4 and (H * W) % 4 == 0 (e.g. 210 x 126, 434 x 252) and one
 * warp's strip of the image in shared memory (fails only for widths near 4096 that are not a multiple of 4);
 * other sizes take the brute-force path, with identical results.
 * May grow library-owned scratch on first use of a larger (n_worlds, H, W) — a device synchronisation and a
 * cudaMalloc —: call gp_reserve first (or warm up) where that must not happen inside the step. */
int gp_render_batch(gp_ctx *ctx, int world_begin, int n_worlds, int agents, int H, int W,
                    float fov_rad, uint8_t *d_class, int32_t *d_instance, float *d_depth,
                    uint8_t *d_rgb, void *stream);

/* Sizes the library-owned per-view scratch (list headers and lists of the cull) for render calls of up to n_worlds worlds
 * with the current rig, and opts the render kernels into the shared memory an H x W image needs.  After it,
 * gp_render_batch with n_worlds' <= n_worlds at that image size allocates nothing and does not synchronise the device.
 * Synchronises the device if it has to grow the scratch.  Call it again after gp_camera_rig_set changed the number of
 * cameras.  GP_ERR_STATE before gp_scene_upload, GP_ERR_RANGE if n_worlds exceeds the scene, GP_ERR_NOMEM. */
int gp_reserve(gp_ctx *ctx, int n_worlds, int H, int W);

/* ---- rendering without any allocation ----------------------------------------------------------------------------
 *
 * Who this is for.  Every other render call needs a gp_ctx, and a gp_ctx owns device memory that the library takes from
 * cudaMalloc (gp_create, gp_scene_upload, the first gp_render_batch of a shape).  Some users of a simulator step cannot
 * accept that:
 *   - a training process whose framework has already claimed all of HBM for its own pool (a caching allocator that grew to
 *     the card's limit, or one told to pre-reserve it): a cudaMalloc from a third-party library then simply fails;
 *   - a latency-bound actor or evaluation loop: cudaMalloc and cudaFree stall the whole device while they run, so one late
 *     allocation in the renderer shows up as a hitch in every other stream of the process;
 *   - a deployment that accounts for each byte of device memory up front and forbids libraries from allocating behind it.
 * gp_render_static serves those.  It takes the scene as device memory the caller already has, renders every view of it
 * (steps a1-a9, the default front camera) into caller-owned planes, and keeps its intermediates - the shading table, the
 * view headers and the per-view primitive lists that the cull writes and the render pass reads - in one fixed array that is
 * part of the library image.  It never calls cudaMalloc, cudaFree or any routine that allocates, and it creates no context.
 *
 * The price is a fixed size.  The array is 9 535 488 bytes (about 9.1 MiB) and exists on every GPU of a process that loads
 * libgp.so, from load until exit, whether this function is called or not.  It bounds the scene:
 *     views   = n_worlds * agents_per_world                      <= GP_STATIC_MAX_VIEWS
 *     records = n_worlds * (agents_per_world + quads_per_world)  <= GP_STATIC_MAX_PRIMS
 *     slots   = views * (agents_per_world + quads_per_world)     <= GP_STATIC_MAX_ENTRIES
 * (16 worlds x 32 agents + 120 quads, or 4 worlds of the paper-scale shape, fit).  Anything larger is refused with
 * GP_ERR_LIMIT before a single launch; split the scene by worlds or use a gp_ctx.
 *
 * Arguments
 *   cuda_device  the device d_prims and the planes live on; must be sm_100 (GP_ERR_ARCH)
 *   desc         HOST, read before the call returns.  n_worlds, agents_per_world, quads_per_world and the constants as for
 *                gp_scene_upload
 *   d_prims      DEVICE [n_worlds][agents_per_world + quads_per_world] gp_prim, 16-byte aligned, agents first in each
 *                world.  Read only; NOT validated (the host never sees it): cls is masked to 0..7 and spheres are drawn
 *   d_pitch_cs   DEVICE [n_worlds][agents_per_world][2] = (cos p, sin p), 8-byte aligned, or NULL for pitch 0
 *   H, W, fov_rad, d_class, d_instance, d_depth, d_rgb   exactly as for gp_render_batch, with one restriction: only image
 *                sizes of the fast path (W >= 4, (H * W) % 4 == 0, one strip within shared memory); others are GP_ERR_ARG
 * The result is the same, bit for bit, as gp_scene_upload + gp_cameras_set + gp_render_batch on the same records.
 *
 * Rules of use
 *   - The first call on each device does a one-off set-up with that device current: it asks the runtime where the array
 *     lives on that device and checks the architecture.  Make that first call outside any stream capture, and before the
 *     part of the program that must not be disturbed.
 *   - All calls on one device share the one array, and it keeps what the previous call left in it.  Nothing in it has to
 *     start at zero - every header and every list slot that is read was written earlier in the same call - and the
 *     headers of the call's views are cleared first all the same, so stale lengths can never be picked up.  Because the
 *     array is shared, two calls must not overlap on the GPU: issue them on one stream, or order the streams with
 *     events.  Calls that run concurrently race on the lists and the planes of both are undefined.  The same holds for
 *     two host threads calling at once on one device.
 *   - Work is enqueued on `stream`; the call does not synchronise.
 * Errors: GP_ERR_ARG, GP_ERR_ALIGN, GP_ERR_LIMIT, GP_ERR_ARCH, GP_ERR_CUDA; all but the last write nothing. */
#define GP_STATIC_MAX_VIEWS   4096
#define GP_STATIC_MAX_PRIMS   32768
#define GP_STATIC_MAX_ENTRIES 131072
int gp_render_static(int cuda_device, const gp_scene_desc *desc, const gp_prim *d_prims, const float *d_pitch_cs,
                     int H, int W, float fov_rad, uint8_t *d_class, int32_t *d_instance, float *d_depth,
                     uint8_t *d_rgb, void *stream);

/* End-to-end variant with HOST buffers: copies h_pose (HOST [Wn][A][4], may be NULL = keep poses) to the
 * device, updates the agents, renders worlds [world_begin, world_begin+n_worlds) in chunks through
 * library-owned device staging and copies the planes (same layouts as above) back to the HOST buffers.
 * Any of the four plane pointers may be NULL (not all): that plane is not copied back — the path is bound by
 * the host link (PCIe), so a consumer that needs e.g. only depth moves a third of the bytes.  Synchronises
 * `stream` before returning.  Pinned host memory is faster but not required. */
int gp_render_batch_host(gp_ctx *ctx, const float *h_pose, int world_begin, int n_worlds, int agents,
                         int H, int W, float fov_rad, uint8_t *h_class, int32_t *h_instance,
                         float *h_depth, uint8_t *h_rgb, void *stream);

/* ---- the step either side of the render --------------------------------------------------- */

/* Limits of the jerk-actuated kinematic bicycle ("accelerations clipped to g-force limits, speed clipped
 * to the speed limit, and the steering angle and its rate bounded"; the paper gives no numbers: caller's choice). */
typedef struct {
    float dt;               /* step, s (the paper simulates at 0.1 s)                                  */
    float a_lon_max;        /* |longitudinal acceleration| limit, m/s^2                                */
    float a_lat_max;        /* |lateral acceleration| limit, m/s^2                                     */
    float v_max;            /* speed limit, m/s: speed is clipped to [0, v_max] (no reversing)         */
    float steer_max;        /* |steering angle| limit, rad; below pi/2 (GP_ERR_ARG otherwise)          */
    float steer_rate_max;   /* |steering rate| limit, rad/s                                            */
    float v_eps;            /* the curvature demand a_lat / v^2 uses max(v, v_eps), m/s (> 0)          */
    float extent;           /* > 0: positions wrap onto the torus [-extent/2, extent/2); 0: no wrap    */
} gp_dyn_params;

/* One simulation step of every agent, on the device (DESIGN.md "Dynamics contract" D1-D6), fused with
 * the pose update a0 of gp_agents_update:
 *   d_action DEVICE int32 [Wn][A]: one of the twelve actions, = 3 * i_lon + i_lat with longitudinal jerk
 *            {-15, -4, 0, 4}[i_lon] and lateral jerk {-4, 0, 4}[i_lat] m/s^3; other values leave the agent untouched,
 *            and so does an agent record of zero length (hx == 0: it has no wheelbase)
 *   d_state  DEVICE fp32 [Wn][A][8], in / out: speed v, a_lon, a_lat, steering angle, heading psi in [-pi, pi), 3 unused
 *   d_pose   DEVICE fp32 [Wn][A][4], in / out: (cx, cy, cos psi, sin psi) — the layout gp_agents_update takes
 * Jerks -> accelerations (clipped) -> speed (clipped to [0, v_max]) -> steering angle demanded by a_lat = v^2 kappa with
 * kappa = tan(steer) / L, wheelbase L = 0.6 * vehicle length (2 hx of the agent's record), bounded in rate and
 * magnitude -> heading -> position (new speed and heading; optional torus wrap).  The new poses are also written into
 * the scene (agent records + shading table), so gp_render_batch can follow with no host transfer.
 * The heading is wrapped into [-pi, pi) however far it turned in the step.
 * fp32 arithmetic with atanf / tanf / sincosf.  Both pointers 16-byte aligned. */
int gp_dynamics_step(gp_ctx *ctx, const gp_dyn_params *params, const int32_t *d_action, float *d_state,
                     float *d_pose, void *stream);

/* The vectorised observation O_vec of every agent (DESIGN.md "Observation contract" O1-O3), from the
 * scene as it stands (agent records as last written by gp_agents_update / gp_dynamics_step; statics).  Ego frame of
 * agent i: origin at its box centre, x along its heading, y to its left.
 *   d_state      DEVICE fp32 [Wn][A][8]: only element 0 (signed speed) of each agent is read
 *   d_agent_idx  DEVICE int32 [Wn][A][K]: the K nearest other agents with squared centre distance <= radius^2, ascending
 *                (distance, index); -1 pads.  "the nearest K within 100 m"
 *   d_agent_feat DEVICE fp32 [Wn][A][K][8]: rel x, rel y, length, width, cos and sin of the relative heading, relative
 *                signed speed v_j - v_i, 1; zeros pad
 *   d_road_idx   DEVICE int32 [Wn][A][M]: primitive indices (>= A) of the M nearest road segments — static box records
 *                with hz == 0 — by their centre, within the radius; -1 pads
 *   d_road_feat  DEVICE fp32 [Wn][A][M][8]: rel x, rel y of the centre, length, cos and sin of the segment's direction in
 *                the ego frame, type (= cls), 1, 0; zeros pad
 * K = 0 or M = 0 skips that part (its pointers may then be NULL).  The paper retrieves segments "from a spatial hash";
 * here every segment of the agent's world is examined from shared memory (a few hundred per world), which returns the
 * same set.  All arithmetic is fp32 add / mul / fma in a fixed order: results are bit-exact against the oracle.
 * K, M <= 1024; GP_ERR_ARG if a world's records do not fit shared memory (more than ~6000 primitives per world).
 * Feature pointers 16-byte aligned. */
int gp_observe_vec(gp_ctx *ctx, const float *d_state, int K, int M, float radius, int32_t *d_agent_idx,
                   float *d_agent_feat, int32_t *d_road_idx, float *d_road_feat, void *stream);

/* Calibration probes for the roofline denominators; synchronises `stream`.
 *   GP_PROBE_STORE: a write-only kernel with the render pass's exact store pattern (per 128 pixels: 4-byte stores to the
 *     class plane and the three colour planes, 16-byte stores to the instance and depth planes = 12 B / pixel) over
 *     n_pixels pixels (a multiple of 128) of the caller's DEVICE planes (sized as for gp_render_batch with n_pixels
 *     pixels in all; their content is overwritten).  Result: GB/s.
 *   GP_PROBE_FMA: 8 independent FFMA chains per thread on (SM count) x 8 CTAs x 256 threads, no memory traffic; the plane
 *     pointers and n_pixels are ignored.  Result: TFLOP/s (2 flop per FFMA) at the clock the GPU runs this at.
 *   GP_PROBE_STORE_VIEW: the same store stream with the render pass's CTA -> address mapping: one CTA per view of the
 *     image size of the last gp_render_batch (H * W a multiple of 128; GP_ERR_STATE before any render), n_pixels a
 *     multiple of H * W, colour planes laid out [view][3][H*W].  Result: GB/s.  The gap to GP_PROBE_STORE is what one
 *     CTA per view costs in DRAM locality; k_render is measured against both.
 *   GP_PROBE_RCP: self-check of the render pass's paired reciprocal (C0: 1.0f / x correctly rounded) against
 *     __frcp_rn on all 2^32 bit patterns; the plane pointers and n_pixels are ignored.  Result: the number of bit
 *     patterns whose result differed, summed over the launches (0 = identical).
 * Runs `iters` timed launches after one warm-up; *best = highest rate, *median (may be NULL) = the median.
 * The probes use device words of their own: the counters gp_stats reads are not disturbed. */
enum { GP_PROBE_STORE = 0, GP_PROBE_FMA = 1, GP_PROBE_RCP = 2, GP_PROBE_STORE_VIEW = 3 };
int gp_probe(gp_ctx *ctx, int kind, size_t n_pixels, int iters, uint8_t *d_class, int32_t *d_instance, float *d_depth,
             uint8_t *d_rgb, void *stream, double *best, double *median);

/* Counters of the last gp_render_batch issued with GP_OPT_STATS = 1 (synchronises the device):
 * executed_tests = ray/primitive slab tests actually evaluated, listed_pairs = (view, primitive)
 * pairs that survived the cull.  Either pointer may be NULL. */
int gp_stats(gp_ctx *ctx, uint64_t *executed_tests, uint64_t *listed_pairs);

/* With GP_OPT_TIMING = n > 0 every n-th launch of each kernel is bracketed by CUDA events on the launch
 * stream (n > 1 keeps the event records from spacing out back-to-back launches).  Returns the summed device time (milliseconds) and the number of launches of `kernel`
 * recorded since the last call for that kernel, then forgets them.  Synchronises the device. */
int gp_kernel_time(gp_ctx *ctx, int kernel, double *total_ms, uint64_t *launches);

/* Number of kernel launches the library has issued on this context since creation. */
int gp_launch_count(gp_ctx *ctx, uint64_t *launches);

const char *gp_error_string(int code);

#ifdef __cplusplus
}
#endif
#endif /* GP_H_ */
