/*
 * gx.h -- C ABI of the B200-native batch RGBD rasteriser.
 *
 * The operation is the rendering hot path of Galactic's simulation step: "A single ... renderer instance
 * renders all environments, sharing GPU memory assets across environments. Scene graph updates are
 * communicated from our physics simulation to the ... renderer ... The renderer outputs a single batch
 * observation per camera sensor, essentially a stack of images from each environment in GPU memory. This is
 * directly consumed by PyTorch GPU-based batch DNN inference, without ever copying pixels to the CPU."
 * (section 3.1).  Sensor: 128x128 RGBD, 90-degree FoV head camera (section 4.1).
 * The paper is silent on the per-pixel arithmetic; it is fixed by DESIGN.md section 3 (readings N0-N10).
 *
 * Conventions (N0): right-handed world, +Y up; the camera looks along its local -Z with +X right
 * and +Y up; all 4x4 matrices are row-major with points as columns; image row 0 is the top row; pixel
 * (col i, row j) has its centre at (i + 0.5, j + 0.5).
 *
 * Threading: one call in flight per handle; distinct handles are independent.  No exception crosses this
 * boundary; every entry point returns 0 or a negative GX_ERR_* code and gx_last_error() holds a
 * thread-local message for the last failure.
 */
#ifndef GX_H_
#define GX_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GX_OK 0
#define GX_ERR_INVALID_ARG (-1) /* null pointer, bad size, bad camera */
#define GX_ERR_CUDA (-2)        /* a CUDA runtime call failed; message has the CUDA error string */
#define GX_ERR_OOM (-3)         /* host or device allocation failed */
#define GX_ERR_UNSUPPORTED (-4) /* valid request outside what this build supports (see gx_render_batch) */

#define GX_BACKGROUND_ID 0xFFFFFFFFu
#define GX_MAX_INSTANCES 254 /* K, instance slots per environment */
#define GX_MAX_FRAME 256     /* width and height limit: the box fields of a triangle record are 8 bits */

typedef struct GxScene GxScene; /* opaque; owns the device copies of all meshes and all scratch memory */

/* One indexed triangle mesh in HOST memory.  Read only during gx_create_scene. */
typedef struct {
    const float *positions;  /* [nv*3] float32, object space (static meshes: world space), metres */
    const uint8_t *colors;   /* [nv*3] uint8 RGB per vertex */
    const uint32_t *indices; /* [nt*3] uint32 vertex indices, each < nv */
    uint32_t nv, nt;
} GxMesh;

/* Pinhole camera shared by all environments of a call. */
typedef struct {
    int32_t width, height; /* pixels; multiples of 16; each <= GX_MAX_FRAME */
    float fx, fy;          /* NDC focal lengths: fy = 1/tan(fovy/2), fx = fy*height/width; 90 deg square: 1 */
    float znear, zfar;     /* metres, 0 < znear < zfar; fragments with view depth > zfar are dropped */
} GxCamera;

/*
 * gx_create_scene -- upload the shared assets once ("sharing GPU memory assets across
 * environments").  static_meshes[s] is the static indoor mesh of scene s (world space); dyn_meshes[m] are
 * the movable-object and robot-link meshes placed per environment by instance transforms.  Every mesh is
 * split into clusters of 256 consecutive triangles, each with its own AABB (frustum-culled per
 * environment); triangle order, and therefore triangle ids, are preserved.
 *   All mesh arrays are HOST pointers and are copied: the caller may free them on return.
 *   cuda_device: ordinal of the device that will own the scene.  *out receives the handle.
 * Errors: INVALID_ARG (null pointers, n_static <= 0, n_dyn < 0, an index >= nv, empty mesh with non-null
 * arrays is allowed), OOM, CUDA.
 */
int gx_create_scene(const GxMesh *static_meshes, int32_t n_static, const GxMesh *dyn_meshes, int32_t n_dyn,
                    int32_t cuda_device, GxScene **out);

/*
 * gx_render_batch -- rasterise RGBD (and optionally triangle ids) for N independent environments.
 * Per pixel: among all post-clip, post-snap triangles of the environment whose integer edge functions
 * cover the pixel centre under the top-left rule and whose depth is <= zfar, the one with the smallest
 * (depth, triangle id, clip sub-index); DESIGN.md section 3 gives every arithmetic step.
 *
 * All array arguments are DEVICE pointers on the scene's device, caller-owned, 16-byte aligned:
 *   env_scene  [N]       int32   static mesh of each environment, in [0, n_static)
 *   cam_pose   [N,16]    float32 camera-to-world, row-major, rigid
 *   inst_mesh  [N,K]     int32   dynamic mesh id in [0, n_dyn), or -1 for an empty slot (may be NULL if K == 0)
 *   inst_xform [N,K,16]  float32 object-to-world, row-major, affine (bottom row ignored)
 *   rgb_out    [N,H,W,3] uint8   may be NULL (depth-only); background (0,0,0)
 *   depth_out  [N,H,W]   float32 planar view-space depth in metres; background 0.0f
 *   id_out     [N,H,W]   uint32  may be NULL; winning triangle id, background GX_BACKGROUND_ID.
 *                                id = j for static triangle j; T_static + sum of nt over earlier non-empty
 *                                slots + j for triangle j of instance slot k.
 *   cuda_stream: a cudaStream_t (NULL = legacy default stream).
 * The call only enqueues work on the stream and returns; outputs are valid in stream order (the zero-copy
 * hand-off of PAPER.md:91).  Scratch inside the handle grows on demand; growing may synchronise the device,
 * steady state does not.  The call may be captured into a CUDA graph (cudaStreamBeginCapture on cuda_stream) once
 * the handle holds its buffers for this shape (gx_reserve, or one plain call): inside a capture it allocates
 * nothing and reads nothing back, and returns UNSUPPORTED if it would have to; replays read the input arrays and
 * write the output arrays the captured call was given.  A graph stays valid for the life of the handle: when a later
 * call makes the handle grow, buffers a captured call used are kept (not freed) until gx_destroy, and the graph goes
 * on rendering with the arena it was captured with.  A call that fails with OOM while growing leaves the handle
 * without an arena but usable: the next call allocates again.  Same inputs give bit-identical outputs, independent of how N is sharded.
 * NaN/Inf inputs and out-of-range env_scene/inst_mesh values are precondition violations: the image is
 * undefined, but no out-of-bounds write occurs for in-range ids.
 * Errors: INVALID_ARG (null handle/camera/required pointer, N <= 0, K < 0, K > GX_MAX_INSTANCES, width or
 * height not a positive multiple of 16, znear <= 0, zfar <= znear), UNSUPPORTED (width or height > 256),
 * OOM, CUDA.
 */
int gx_render_batch(GxScene *scene, const GxCamera *camera, int32_t N, int32_t K, const int32_t *env_scene,
                    const float *cam_pose, const int32_t *inst_mesh, const float *inst_xform, uint8_t *rgb_out,
                    float *depth_out, uint32_t *id_out, void *cuda_stream);

/*
 * gx_render_batch_noalloc -- gx_render_batch for callers that must not enter the CUDA allocator while they render.
 *
 * Who that is: gx_render_batch and gx_reserve obtain the record arena and the per-call tables with cudaMalloc (and
 * give them back with cudaFree when they have to grow).  That is unusable where the renderer is a guest on a device
 * whose memory another component has already claimed -- a simulation worker inside a training process whose tensor
 * allocator holds all remaining device memory, so that a cudaMalloc of the arena fails or takes memory the policy's
 * next batch needs -- and where the render call runs beside other streams (the policy's inference):
 * cudaMalloc and cudaFree wait for the whole device, so one growing render call stalls every stream of the process.
 * Such callers own their inputs and outputs (they pass them here as usual) but have no way to own the renderer's
 * intermediate memory, which has no public layout.
 *
 * What it does instead: the arena and the tables are carved out of one array of GX_NOALLOC_SCRATCH_BYTES bytes that
 * is part of the library's device image (a file-scope __device__ array; every GPU that uses libgx.so holds these
 * bytes from the time the library's kernels are loaded on it until the process exits, whether or not this entry
 * point is ever called).  K1 (cull_kernel) runs as in gx_render_batch with its tables in that array; K2-K5 run as
 * one cooperative kernel, a variant of the tail kernel of gx_render_batch that starts at the first environment and
 * renders the batch in as many waves as the arena left in the array requires.  The images are the same, bit for bit
 * (tests/test_zz_no_alloc.py); a call is slower than gx_render_batch when it needs several waves.
 *
 * Arguments, stream semantics and results exactly as gx_render_batch.  The options "cull", "subcull", "hiz",
 * "occlusion", "occl_area", "big_px" and "ctas_per_sm" apply; "stats", "timing", "pool_bytes" and "arena_slots" do not, and
 * gx_get_stat keeps describing the last gx_render_batch.  The scene handle still comes from gx_create_scene, which
 * allocates (meshes are uploaded once, at start-up, before the device's memory is handed to anyone else).
 *   The call itself uses no cudaMalloc, cudaMallocAsync, cudaFree or other allocating routine, on any path.
 *   Limit: the tables of the call shape (about 150 KB per environment at 128x128 with 25 instance slots; 8 bytes per
 *   pixel plus the work-item lists) and an arena for at least the largest environment the scene can produce
 *   (88 bytes x (4 x (largest static mesh + K x largest dynamic mesh, in triangles) + 64)) must fit
 *   GX_NOALLOC_SCRATCH_BYTES together; e.g. up to about 250 environments of a 50k-triangle scene with 25 slots of
 *   1k-triangle meshes at 128x128.  A shape beyond that returns UNSUPPORTED and the message names the bytes needed
 *   and the bytes there are; nothing is enqueued.
 *   First call on a device: looks up the array's device address and the launch shape of the cooperative kernel for
 *   that device and keeps them for the process's lifetime (no allocation; a few driver queries).  Make that first
 *   call outside any stream capture.
 *   Sharing: every call on a device, from every handle and every thread, uses the same array.  The call clears the
 *   words that must start at zero (control words, the hi-Z pyramid) on cuda_stream itself and overwrites everything
 *   else before reading it, so the previous call's contents never show; but two calls whose GPU work overlaps (two
 *   streams, two threads, two handles) race on the array and give undefined images.  Order them on one stream or
 *   with events.  gx_render_batch does not use the array and may overlap with it.
 * Errors: as gx_render_batch, plus UNSUPPORTED (shape beyond the array; device ordinal >= 64; device without
 * cooperative launch).
 */
#define GX_NOALLOC_SCRATCH_BYTES (64u << 20)
int gx_render_batch_noalloc(GxScene *scene, const GxCamera *camera, int32_t N, int32_t K, const int32_t *env_scene,
                            const float *cam_pose, const int32_t *inst_mesh, const float *inst_xform, uint8_t *rgb_out,
                            float *depth_out, uint32_t *id_out, void *cuda_stream);

/*
 * gx_reserve -- allocate (or grow) everything the handle needs for calls of this shape now, so that the render calls
 * that follow never allocate: the record arena (option "pool_bytes": at most an eighth of the device's memory and
 * 16 GB by default; what does not fit is rendered in further waves) and the per-call tables.  Optional: the first
 * gx_render_batch of a shape does the same.  "arena_bytes" and "scratch_bytes" of gx_get_stat tell what is held.
 * Errors: INVALID_ARG, OOM, CUDA.
 */
int gx_reserve(GxScene *scene, const GxCamera *camera, int32_t N, int32_t K);

/*
 * gx_render_batch_obs -- the same rasterisation, written as the packed observation tensor the policy reads
 * ("directly consumed by PyTorch GPU-based batch DNN inference"; the visual encoder takes RGBD,
 * PAPER.md:141, Table 3).  The paper is silent on the layout and normalisation; N11 fixes them:
 *   obs_out [N,4,H,W] IEEE binary16, DEVICE pointer, 8-byte aligned: planes R, G, B = binary16(c / 255.0f) with c
 *   the uint8 channel of gx_render_batch, plane D = binary16((clamp(depth, depth_min, depth_max) - depth_min) /
 *   (depth_max - depth_min)) with depth the float32 depth of gx_render_batch (background 0.0f, so its D is 0);
 *   all operations float32, conversions round-to-nearest-even.  The packing is fused into the last step of the
 *   raster kernel: no RGB or depth image is written.
 * Other arguments, stream semantics and errors as gx_render_batch; additionally INVALID_ARG if obs_out is NULL
 * or depth_max <= depth_min.
 */
int gx_render_batch_obs(GxScene *scene, const GxCamera *camera, int32_t N, int32_t K, const int32_t *env_scene,
                        const float *cam_pose, const int32_t *inst_mesh, const float *inst_xform, uint16_t *obs_out,
                        float depth_min, float depth_max, void *cuda_stream);

/*
 * gx_render_batch_host -- the same operation with every array argument in HOST memory (pageable or
 * pinned): copies the inputs to the device, renders in three sub-batches (option "host_sub") while the images of
 * the previous sub-batch are copied back on a second stream, and synchronises before returning.  This is the
 * end-to-end entry point bench.py times for its "e2e" figure.
 */
int gx_render_batch_host(GxScene *scene, const GxCamera *camera, int32_t N, int32_t K, const int32_t *env_scene,
                         const float *cam_pose, const int32_t *inst_mesh, const float *inst_xform,
                         uint8_t *rgb_out, float *depth_out, uint32_t *id_out);

/*
 * GxLink, gx_set_robot, gx_update_transforms -- the scene-graph update on the GPU: forward kinematics from the
 * per-environment base pose and joint positions to the link, camera and held-object transforms, written straight
 * into the arrays gx_render_batch reads ("we use forward kinematics to compute the position of the robot's
 * articulated links"; "Scene graph updates are communicated from our physics simulation to the ...
 * renderer"; it replaces the CPU "Render Setup" stage of Table 5).  The paper gives no
 * robot format or arithmetic; N12 fixes both (binary32, own sine / cosine, Rodrigues joints, the affine
 * product order of N2).
 *
 * gx_set_robot: links [n_links] HOST array, copied.  Link l hangs off link parent < l (-1 = the base); origin is the
 *   joint frame in the parent link's frame (3x4 row-major, rigid); joint_type 0 fixed, 1 revolute about, 2 prismatic
 *   along the unit vector axis (joint frame).  camera_link / cam_mount [12]: the link the camera rides on (-1 = the
 *   base) and the camera frame in that link's frame; ee_link: the link that carries a held object (-1 = the base).
 *   Errors: INVALID_ARG (NULL, n_links outside [1, 64], a parent that does not precede its link, a joint type
 *   outside 0..2, link indices out of range), OOM, CUDA.
 * gx_update_transforms: all arrays are DEVICE pointers, caller-owned; rows of 16 floats must be 16-byte aligned.
 *   base_pose  [N,3]     float32 in   x, z, yaw: the base stands on the ground plane y = 0 and turns about +Y
 *   joint_pos  [N,L]     float32 in   one position per link (radians or metres; ignored for fixed joints)
 *   held_slot  [N]       int32   in   instance slot of the object in the gripper, -1 = none; NULL = no held objects
 *   held_xform [N,12]    float32 in   the held object's pose in the end-effector link's frame (3x4); NULL with held_slot
 *   cam_pose   [N,16]    float32 out  camera-to-world of every environment
 *   inst_xform [N,K,16]  float32 i/o  slots link_slot0 .. link_slot0 + L - 1 receive the link transforms, slot
 *                                     held_slot[n] the held object's; every other slot is left as it is
 *   The call only enqueues one kernel on cuda_stream; a gx_render_batch enqueued after it on the same stream sees
 *   the new transforms.  Errors: INVALID_ARG (no robot set, NULL arrays, N <= 0, link slots outside [0, K)), CUDA.
 */
typedef struct {
    int32_t parent;
    int32_t joint_type;
    float axis[3];
    float origin[12];
} GxLink;
int gx_set_robot(GxScene *scene, const GxLink *links, int32_t n_links, int32_t camera_link, const float *cam_mount,
                 int32_t ee_link);
int gx_update_transforms(GxScene *scene, int32_t N, int32_t K, int32_t link_slot0, const float *base_pose,
                         const float *joint_pos, const int32_t *held_slot, const float *held_xform, float *cam_pose,
                         float *inst_xform, void *cuda_stream);

/*
 * GxColumnGrid, GxSphere, gx_set_collision_world, gx_collide_batch -- the batch collision queries of the kinematic
 * simulator on the GPU ("This new candidate pose for the robot is tested for overlap (penetration) with
 * the environment"; PAPER.md:111-119 and Appendix G): every sphere of the robot against the static
 * scene's column grid of its radius and against the oriented boxes of the resting movable objects.  The paper gives
 * the structures but no layout or arithmetic; N13 fixes both.  Its layer cache and its four offset regular
 * grids are accelerations of the same answer for a CPU; here every sphere tests all boxes of its environment.
 *
 * gx_set_collision_world: HOST arrays, copied.  grids [n_static * n_radii], grid (scene s, radius class c) at
 *   s * n_radii + c: columns in the XZ plane at `spacing` (0.03 m in the paper), column (ix, iz) at
 *   col_off[iz * nx + ix] .. col_off[iz * nx + ix + 1] of `layers`, a layer = (lo, hi), the heights the CENTRE of a
 *   sphere of that radius may take (both inclusive).  radii [n_radii]: the sphere-radius working set ({0.015, 0.05,
 *   0.12} in the paper).  spheres [n_spheres]: link index (>= 0), radius class, centre in the link's frame; link -1
 *   puts the sphere on the grasped object ("the robot (and the current grasped object, if any)"): its
 *   centre is in that object's frame and it moves with inst_xform[n][held_slot[n]].
 *   Errors: INVALID_ARG, UNSUPPORTED (more than 2^32 columns or layers), OOM, CUDA.
 * gx_collide_batch: DEVICE arrays.  Sphere centres are W_link * centre with W_link = inst_xform[n][link_slot0 + link]
 *   (what gx_update_transforms wrote); for a sphere with link -1, W = inst_xform[n][held_slot[n]], and where nothing
 *   is held (held_slot NULL, or held_slot[n] outside [0, K)) that sphere reports 0 and -1.  The box of instance slot k is the object-space bounding box of its mesh
 *   under inst_xform[n][k], which must be rigid.
 *   out_static [N, n_spheres] uint8: 1 if the sphere is in obstructed space of its column grid or outside the grid.
 *   out_object [N, n_spheres] int32: the lowest slot in [obj_slot0, obj_slot0 + n_obj) whose box the sphere overlaps
 *   (distance from the centre to the box <= radius), skipping empty slots and held_slot[n] (NULL = nothing held); -1
 *   if none.  Enqueues one kernel on cuda_stream.  Errors: INVALID_ARG (no collision world, NULL arrays, slots outside
 *   [0, K)), CUDA.
 */
typedef struct {
    float x0, z0;
    float spacing;
    int32_t nx, nz;
    const uint32_t *col_off;
    const float *layers;
} GxColumnGrid;
typedef struct {
    int32_t link;
    int32_t radius_class;
    float centre[3];
} GxSphere;
int gx_set_collision_world(GxScene *scene, const GxColumnGrid *grids, int32_t n_radii, const float *radii,
                           const GxSphere *spheres, int32_t n_spheres);
int gx_collide_batch(GxScene *scene, int32_t N, int32_t K, const int32_t *env_scene, const int32_t *inst_mesh,
                     const float *inst_xform, int32_t link_slot0, int32_t obj_slot0, int32_t n_obj,
                     const int32_t *held_slot, uint8_t *out_static, int32_t *out_object, void *cuda_stream);

/*
 * gx_set_option -- tuning / verification switches of a handle.  Unknown names and out-of-range values return
 * INVALID_ARG.  Every switch leaves the images bit-identical (tested); they only move time around.
 *   "cull"         0|1 (1)   per-environment frustum culling of clusters (K1).
 *   "subcull"      0|1 (1)   the same test for every run of 32 triangles of a visible cluster.
 *   "hiz"          0|1 (1)   hi-Z rejection (in the tiles, and with it the occluder scheme).
 *   "occlusion"    -1|0|1 (-1) occluder scheme: the runs whose triangles are big on screen go through
 *                            geometry / bin / raster first, the others are culled against the hi-Z values that
 *                            leaves (per run and per triangle) and follow in a second phase.  -1 = automatic: on
 *                            for frames of at least 4096 pixels.
 *   "occl_area"    (64)      screen-box pixels per triangle from which a run counts as big.
 *   "big_px"       1..32 (24) records whose pixel box is at least this wide or high take the large (block) path.
 *   "pool_bytes"   budget of the record arena, which bounds the environments per wave; 0 = an eighth of the
 *                            device's memory, at most 16 GB.
 *   "arena_slots"  force the arena size in record slots (tests: several waves); 0 = automatic.
 *   "host_sub"     environments per sub-batch of gx_render_batch_host; 0 = a third of the batch.
 *   "ctas_per_sm"  0..8 (0 = as many as fit) CTAs per SM of the persistent geometry and raster kernels, for callers
 *                            that run other kernels beside the renderer.
 *   "bin_threads"  0|256|512 (0 = 512) threads per CTA of the bin kernel.
 *   "max_rounds"   >= 0 (0 = no limit) rounds of stage kernels the host launches per call; with several waves the
 *                            host launches one round per wave the previous call needed and the cooperative tail kernel
 *                            renders what is left, so 1 sends every wave after the first to the tail kernel (tests).
 *   "stats"        0|1 (0)   count what gx_get_stat reports (slower kernels).
 *   "timing"       0|1 (0)   1 starts (and resets), 0 stops recording CUDA events around every kernel of
 *                            subsequent gx_render_batch calls on their stream.
 */
int gx_set_option(GxScene *scene, const char *name, int64_t value);

/*
 * gx_get_stat -- counters of the most recent gx_render_batch on this handle ("stats" = 1); synchronises the
 * stream the call ran on.  Names: "clusters_tested", "clusters_drawn", "triangles_in" (triangles of drawn
 * runs), "triangles_raster" (survived clip, zero-area and pixel-centre bounding-box rejection and the hi-Z test of
 * the second phase), "triangles_hidden", "subclusters_hidden" (dropped by the hi-Z tests of the second phase),
 * "fragments" (pixel-centre hits that reached the depth test), "records_occluded" (references dropped by hi-Z in
 * the tiles), "blocks_drawn", "large_records", "large_draws", "tile_refs", "waves", "sum_slots", "max_env_slots"
 * (record slot bounds), "bad_ids" (out-of-range mesh ids treated as empty slots), "launches" (kernels launched by
 * the call), "arena_bytes", "scratch_bytes", "bound_violations" (the kernels' own index checks in the stats build: always 0).
 * With "timing": "timed_calls" and "ns_cull", "ns_geom", "ns_bin", "ns_raster", "ns_tail" = nanoseconds spent in
 * each kernel class, summed over the calls since timing was started.
 * Unknown names return INVALID_ARG; *out receives the value.
 */
int gx_get_stat(GxScene *scene, const char *name, int64_t *out);

/* gx_destroy -- free the handle and everything it owns.  NULL is allowed. */
void gx_destroy(GxScene *scene);

/* gx_last_error -- thread-local, NUL-terminated message for the last non-zero return on this thread. */
const char *gx_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GX_H_ */
