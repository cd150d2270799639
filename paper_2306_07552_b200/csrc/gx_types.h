// gx_types.h -- device-side data layout shared by the host API (gx_api.cu) and the kernels (gx_pipeline.cuh).
// Product code: nothing here is shared with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

// A mesh is cut into clusters of GX_CLUSTER_TRIS consecutive triangles (the culling unit, one AABB each;
// BASELINE.json north_star (1)).  A cluster is stored as 1..4 batches: a batch is a run of consecutive
// triangles that references at most GX_VCAP unique vertices, so that one warp can stage the batch's
// transformed vertices in shared memory and triangles can index them with 8 bits.  Well-indexed meshes
// (0.5-0.6 vertices per triangle) give exactly one batch per cluster; a non-indexed soup gives 85-triangle
// batches.  Triangle order is never changed, so triangle id = position in the caller's index array.
constexpr int GX_CLUSTER_TRIS = 256;
constexpr int GX_VCAP = 256;            // unique vertices per batch (8-bit local indices)
constexpr int GX_SUBS_PER_BATCH = GX_CLUSTER_TRIS / 32;   // sub-cluster = 32 consecutive triangles = one warp pass
constexpr int GX_MAX_BATCH_PER_CLUSTER = 4;  // 85 soup triangles need 255 vertices -> ceil(256/85) = 4

struct __align__(16) GxBatchDev {
    uint32_t vert_off;   // first entry in GxSceneDev::verts
    uint32_t tri_off;    // first entry in GxSceneDev::tris
    uint32_t nv_nt;      // nv | nt << 16
    uint32_t first_tri;  // mesh-local id of the batch's first triangle
};

struct __align__(16) GxClusterDev {
    float bmin[3];
    uint32_t batch_off;  // first batch (global index)
    float bmax[3];
    uint32_t nbatch;
};

struct __align__(16) GxMeshDev {
    uint32_t cluster_off, ncluster, nt, pad;
};

// What every stage of one gx_render_batch call needs; passed by value inside PipeParams (gx_pipeline.cuh).
struct GxParams {
    // scene (device)
    const float4 *verts;          // x, y, z, rgba8 bits; per batch contiguous
    const uchar4 *tris;           // three batch-local vertex indices; per batch contiguous
    const GxBatchDev *batches;
    const GxClusterDev *subs;     // [batch][GX_SUBS_PER_BATCH] AABB of each run of 32 consecutive triangles of a batch
    const GxClusterDev *clusters;
    const GxMeshDev *meshes;      // static meshes first, then dynamic
    int32_t n_static, n_dyn;
    // call
    int32_t N, K, W, H;
    float fx, fy, znear, zfar;
    const int32_t *env_scene;
    const float *cam_pose;
    const int32_t *inst_mesh;
    const float *inst_xform;
    uint8_t *rgb;
    float *depth;
    uint32_t *id;
    uint16_t *obs;                // [N,4,H,W] binary16 packed observation (N11), or NULL
    float obs_dmin, obs_dmax, obs_range;   // depth channel = (clamp(depth, dmin, dmax) - dmin) / range, range = dmax - dmin
    unsigned long long *stats;    // [GX_NSTAT], only touched by the STATS instantiations
    int32_t cull;                 // 0 = draw every cluster (verification)
};

enum { GX_STAT_CLUSTERS_TESTED = 0, GX_STAT_CLUSTERS_DRAWN, GX_STAT_TRIS_IN, GX_STAT_TRIS_RASTER,
       GX_STAT_FRAGMENTS, GX_STAT_RECORDS_OCCLUDED, GX_STAT_BLOCKS_DRAWN, GX_STAT_REFS, GX_STAT_TRIS_HIDDEN,
       GX_STAT_SUBS_HIDDEN, GX_STAT_LARGE, GX_STAT_LARGE_DRAWS, GX_STAT_VIOLATIONS, GX_NSTAT };
