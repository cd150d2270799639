// gx_api.cu -- host side of the C ABI declared in include/gx.h: scene upload (clustering), launch, errors.
// Product code.  Nothing here includes, links or calls anything under oracle/.
#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/gx.h"
#include "gx_pipeline.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define GX_CUDA(call)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? GX_ERR_OOM : GX_ERR_CUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                   \
    } while (0)

struct DeviceGuard {   // make the scene's device current for the duration of a call
    int prev = -1;
    bool ok = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) return;
        ok = prev == dev || cudaSetDevice(dev) == cudaSuccess;
        if (prev == dev) prev = -1;
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

template <typename T>
struct DevBuf {
    T *p = nullptr;
    size_t n = 0;
    int reserve(size_t want) {   // grow only; contents are not kept
        if (want <= n) return GX_OK;
        if (p) cudaFree(p);
        p = nullptr;
        n = 0;
        GX_CUDA(cudaMalloc(&p, want * sizeof(T)));
        n = want;
        return GX_OK;
    }
    void release() {
        if (p) cudaFree(p);
        p = nullptr;
        n = 0;
    }
};

}  // namespace

struct GxScene {
    int device = 0;
    int num_sms = 0;
    int n_static = 0, n_dyn = 0;
    float4 *verts = nullptr;
    uchar4 *tris = nullptr;
    GxBatchDev *batches = nullptr;
    GxClusterDev *subs = nullptr;
    GxClusterDev *clusters = nullptr;
    GxMeshDev *meshes = nullptr;
    std::vector<uint32_t> mesh_nt;      // host copy, for id-range validation
    uint32_t max_dyn_nt = 0, max_static_nt = 0;
    uint32_t max_nbatch = 1;            // largest number of batches in any cluster
    uint32_t max_static_batches = 0, max_dyn_batches = 0;   // largest number of batches in any static / dynamic mesh
    int max_smem_optin = 0;
    unsigned int *env_counter = nullptr;
    unsigned long long *stats = nullptr;   // device [GX_NSTAT]
    int opt_cull = 1;
    int opt_stats = 0;
    int last_chunk_n = 0;               // environments in the last chunk of the last two-kernel call
    int opt_path = 0;                   // 0 = two-kernel path (geometry -> records -> raster), 1 = single kernel
    int64_t opt_pool_slots = 0;         // narrow record slots per environment; 0 = max(4096, 4*W*H)
    int64_t opt_pool_bytes = 0;         // record pool budget; 0 = 8 GB
    int opt_big_slots = 512, opt_chunk_slots = 128;   // raster pass B (gx_pipeline.cuh)
    DevBuf<uint4> pool;                 // triangle records of one chunk of environments
    DevBuf<unsigned long long> frames;  // frame keys between the two raster phases
    // kernel timing (option "timing"): CUDA events recorded on the caller's stream around every kernel class
    int opt_timing = 0;
    std::vector<cudaEvent_t> t_ev;      // recorded marks, in order
    std::vector<int> t_kind;            // what ran before the mark: 0 = start of a pass, 1 cull, 2 geom, 3 order, 4 raster, 5 fallback
    size_t t_used = 0;
    int t_calls = 0;
    int opt_subcull = 1;                // geometry kernel: frustum (and hi-Z) test per 32-triangle sub-cluster
    int opt_bands = 0;                  // raster bands per frame; 0 = automatic
    int opt_occlusion = 1;              // occluder scheme: 0 off, 2 or 3 passes, 1 = automatic
    int opt_occl_area = 64;              // occluder scheme: sub-clusters with >= this many screen-box pixels per triangle go first
    int opt_occluder_pct = 50;          // share of the visible clusters (nearest first) drawn in the occluder phase
    // pool sizing from history: the largest record counts any raster task of earlier calls produced
    uint32_t *d_maxrec = nullptr, *h_maxrec = nullptr;   // device [2]; pinned host [2]
    cudaEvent_t ev_maxrec = nullptr;
    bool maxrec_pending = false;
    uint32_t hist_n = 0, hist_w = 0;
    DevBuf<uint32_t> pipe_scratch;      // counters[4] | cnt[2*chunk] | env_flag[chunk]
    int last_launches = 0;
    cudaStream_t last_stream = nullptr;
    // staging for gx_render_batch_host
    DevBuf<int32_t> h_env_scene, h_inst_mesh;
    DevBuf<float> h_cam_pose, h_inst_xform, h_depth;
    DevBuf<uint8_t> h_rgb;
    DevBuf<uint32_t> h_id;
    cudaStream_t host_stream = nullptr, copy_stream = nullptr;
    cudaEvent_t ev_sub = nullptr;
};

namespace {

// Cut one mesh into clusters of GX_CLUSTER_TRIS consecutive triangles and batches of <= GX_VCAP unique
// vertices (gx_types.h).  Vertices are copied per batch in first-use order with the colour packed into .w.
int build_mesh(const GxMesh &m, std::vector<float4> &verts, std::vector<uchar4> &tris, std::vector<GxBatchDev> &batches,
               std::vector<GxClusterDev> &subs, std::vector<GxClusterDev> &clusters, GxMeshDev &out) {
    out.cluster_off = (uint32_t)clusters.size();
    out.nt = m.nt;
    out.pad = 0;
    std::vector<int32_t> local(m.nv, -1);
    std::vector<uint32_t> touched;
    touched.reserve(GX_VCAP);
    for (uint32_t t0 = 0; t0 < m.nt; t0 += GX_CLUSTER_TRIS) {
        const uint32_t t1 = std::min<uint32_t>(t0 + GX_CLUSTER_TRIS, m.nt);
        GxClusterDev c;
        c.batch_off = (uint32_t)batches.size();
        c.nbatch = 0;
        for (int k = 0; k < 3; ++k) { c.bmin[k] = 3.0e38f; c.bmax[k] = -3.0e38f; }
        uint32_t t = t0;
        while (t < t1) {
            GxBatchDev b;
            b.vert_off = (uint32_t)verts.size();
            b.tri_off = (uint32_t)tris.size();
            b.first_tri = t;
            uint32_t nv = 0, nt = 0;
            touched.clear();
            for (; t < t1; ++t, ++nt) {
                uint32_t idx[3];
                int fresh = 0;
                for (int k = 0; k < 3; ++k) {
                    idx[k] = m.indices[3 * (size_t)t + k];
                    if (idx[k] >= m.nv) return fail(GX_ERR_INVALID_ARG, "triangle %u references vertex %u >= nv %u", t, idx[k], m.nv);
                    if (local[idx[k]] < 0 && (k < 1 || idx[k] != idx[0]) && (k < 2 || idx[k] != idx[1])) ++fresh;
                }
                if (nv + fresh > (uint32_t)GX_VCAP) break;
                uchar4 li;
                unsigned char *lp = &li.x;
                for (int k = 0; k < 3; ++k) {
                    if (local[idx[k]] < 0) {
                        local[idx[k]] = (int32_t)nv++;
                        touched.push_back(idx[k]);
                        const float *p = m.positions + 3 * (size_t)idx[k];
                        const uint8_t *col = m.colors + 3 * (size_t)idx[k];
                        const uint32_t rgba = (uint32_t)col[0] | ((uint32_t)col[1] << 8) | ((uint32_t)col[2] << 16);
                        float4 v;
                        v.x = p[0]; v.y = p[1]; v.z = p[2];
                        memcpy(&v.w, &rgba, 4);
                        verts.push_back(v);
                        for (int a = 0; a < 3; ++a) {
                            c.bmin[a] = std::min(c.bmin[a], p[a]);
                            c.bmax[a] = std::max(c.bmax[a], p[a]);
                        }
                    }
                    lp[k] = (unsigned char)local[idx[k]];
                }
                li.w = 0;
                tris.push_back(li);
            }
            b.nv_nt = nv | (nt << 16);
            // sub-clusters: AABB of every run of 32 consecutive triangles of the batch
            for (uint32_t k = 0; k < (uint32_t)GX_SUBS_PER_BATCH; ++k) {
                GxClusterDev sb;
                uint32_t vlo = 0xFFFFu, vhi = 0;   // batch-local vertex index range of the sub-cluster's triangles
                for (int a = 0; a < 3; ++a) { sb.bmin[a] = 3.0e38f; sb.bmax[a] = -3.0e38f; }
                for (uint32_t tt = b.first_tri + 32 * k; tt < std::min(b.first_tri + 32 * (k + 1), b.first_tri + nt); ++tt)
                    for (int kk = 0; kk < 3; ++kk) {
                        const uint32_t lv = (uint32_t)local[m.indices[3 * (size_t)tt + kk]];
                        vlo = std::min(vlo, lv);
                        vhi = std::max(vhi, lv);
                        const float *pp = m.positions + 3 * (size_t)m.indices[3 * (size_t)tt + kk];
                        for (int a = 0; a < 3; ++a) {
                            sb.bmin[a] = std::min(sb.bmin[a], pp[a]);
                            sb.bmax[a] = std::max(sb.bmax[a], pp[a]);
                        }
                    }
                sb.batch_off = vlo;   // (fields reused: first and last vertex the sub-cluster references)
                sb.nbatch = vhi;
                subs.push_back(sb);
            }
            for (uint32_t v : touched) local[v] = -1;
            batches.push_back(b);
            ++c.nbatch;
        }
        clusters.push_back(c);
    }
    out.ncluster = (uint32_t)clusters.size() - out.cluster_off;
    return GX_OK;
}

template <typename T>
int upload(T *&dst, const std::vector<T> &src) {
    const size_t n = std::max<size_t>(src.size(), 1);
    GX_CUDA(cudaMalloc(&dst, n * sizeof(T)));
    if (!src.empty()) GX_CUDA(cudaMemcpy(dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return GX_OK;
}

struct LaunchPlan {
    int warps, minb;
    size_t smem;
    int grid;
};

template <int WARPS, int MINB>
int launch(const GxScene *sc, const GxParams &P, size_t smem, cudaStream_t stream, bool stats) {
    auto kern = stats ? gx::render_kernel<WARPS, MINB, true> : gx::render_kernel<WARPS, MINB, false>;
    GX_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    GX_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, WARPS * 32, smem));
    if (per_sm < 1) return fail(GX_ERR_UNSUPPORTED, "kernel does not fit: %zu bytes of shared memory", smem);
    const int grid = std::min(P.N, sc->num_sms * per_sm);
    kern<<<grid, WARPS * 32, smem, stream>>>(P);
    GX_CUDA(cudaGetLastError());
    return GX_OK;
}


// single-kernel path (gx_kernels.cuh): small frames (<= 32 KB of keys) use 8-warp CTAs, several per SM; big
// frames one CTA per SM with as many warps as the rest of the 227 KB of shared memory holds staging for.
int launch_single(const GxScene *sc, const GxParams &P, cudaStream_t stream, bool st) {
    const int K = P.K;
    const bool small_frame = (size_t)P.W * P.H * 8 <= 32768;
    const size_t cap = (size_t)sc->max_smem_optin - 256;   // static shared memory of the kernel
    if (small_frame) return launch<8, 2>(sc, P, gx::kernel_smem_bytes(P.W, P.H, K, 8), stream, st);
    if (gx::kernel_smem_bytes(P.W, P.H, K, 16) <= cap) return launch<16, 1>(sc, P, gx::kernel_smem_bytes(P.W, P.H, K, 16), stream, st);
    if (gx::kernel_smem_bytes(P.W, P.H, K, 12) <= cap) return launch<12, 1>(sc, P, gx::kernel_smem_bytes(P.W, P.H, K, 12), stream, st);
    return launch<8, 1>(sc, P, gx::kernel_smem_bytes(P.W, P.H, K, 8), stream, st);
}

template <int WARPS, int MINB, int PHASE>
int launch_raster(const GxScene *sc, const gx::PipeParams &PP, cudaStream_t stream, bool stats) {
    auto kern = stats ? gx::raster_kernel<WARPS, MINB, PHASE, true> : gx::raster_kernel<WARPS, MINB, PHASE, false>;
    const size_t smem = gx::raster_smem_bytes(PP.g.W, PP.bh, WARPS);
    GX_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    GX_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, WARPS * 32, smem));
    if (per_sm < 1) return fail(GX_ERR_UNSUPPORTED, "raster kernel does not fit: %zu bytes of shared memory", smem);
    kern<<<std::min(PP.g.N * PP.bands, sc->num_sms * per_sm), WARPS * 32, smem, stream>>>(PP);
    GX_CUDA(cudaGetLastError());
    return GX_OK;
}

// timing mark: an event on the stream; the time since the previous mark belongs to kernel class `kind`
int mark(GxScene *sc, cudaStream_t stream, int kind) {
    if (!sc->opt_timing || sc->t_used >= 8192) return GX_OK;
    if (sc->t_used == sc->t_ev.size()) {
        cudaEvent_t e;
        GX_CUDA(cudaEventCreate(&e));
        sc->t_ev.push_back(e);
        sc->t_kind.push_back(0);
    }
    sc->t_kind[sc->t_used] = kind;
    GX_CUDA(cudaEventRecord(sc->t_ev[sc->t_used], stream));
    ++sc->t_used;
    return GX_OK;
}

// one pass of the pipeline (gx_pipeline.cuh): cull kernel, geometry kernel, raster order, raster kernel.
// PHASE 0 = everything in one pass; 1 = occluder phase; 2 = the rest, culled against the occluder phase's hi-Z.
template <int PHASE>
int launch_pass(GxScene *sc, const gx::PipeParams &PP, cudaStream_t stream, bool stats) {
    int rc;
    if ((rc = mark(sc, stream, 0)) != GX_OK) return rc;
    constexpr int GW = 8, CP = PHASE >= 2 ? 2 : 1;
    const size_t csmem = gx::env_smem_bytes(PP.g.K);
    // one CTA per environment: 4 warps for small scenes, 16 where an environment has thousands of sub-clusters to test
    if ((size_t)sc->max_static_batches + (size_t)PP.g.K * sc->max_dyn_batches > 512) {
        auto ck = stats ? gx::cull_kernel<16, CP, true> : gx::cull_kernel<16, CP, false>;
        ck<<<PP.g.N, 16 * 32, csmem, stream>>>(PP);
    } else {
        auto ck = stats ? gx::cull_kernel<4, CP, true> : gx::cull_kernel<4, CP, false>;
        ck<<<PP.g.N, 4 * 32, csmem, stream>>>(PP);
    }
    GX_CUDA(cudaGetLastError());
    if ((rc = mark(sc, stream, 1)) != GX_OK) return rc;
    auto gk = stats ? gx::geom_kernel<GW, true> : gx::geom_kernel<GW, false>;
    const size_t gsmem = (size_t)GW * gx::GEOM_WARP_SMEM;
    GX_CUDA(cudaFuncSetAttribute(gk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gsmem));
    int per_sm = 0;
    GX_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, gk, GW * 32, gsmem));
    if (per_sm < 1) return fail(GX_ERR_UNSUPPORTED, "geometry kernel does not fit: %zu bytes of shared memory", gsmem);
    gk<<<sc->num_sms * per_sm, GW * 32, gsmem, stream>>>(PP);
    GX_CUDA(cudaGetLastError());
    if ((rc = mark(sc, stream, 2)) != GX_OK) return rc;
    gx::order_kernel<<<1, 1024, 0, stream>>>(PP, PHASE >= 2 ? 1 : 0);
    GX_CUDA(cudaGetLastError());
    if ((rc = mark(sc, stream, 3)) != GX_OK) return rc;
    // one band of 64-bit keys per CTA: the smaller the band, the more CTAs share an SM (32 warps per SM in all cases)
    const size_t band_bytes = (size_t)PP.g.W * PP.bh * 8;
    if (band_bytes <= 32768) rc = launch_raster<8, 4, PHASE>(sc, PP, stream, stats);
    else if (band_bytes <= 65536) rc = launch_raster<16, 2, PHASE>(sc, PP, stream, stats);
    else rc = launch_raster<32, 1, PHASE>(sc, PP, stream, stats);
    if (rc != GX_OK) return rc;
    return mark(sc, stream, 4);
}

}  // namespace

extern "C" {

const char *gx_last_error(void) { return g_err; }

int gx_create_scene(const GxMesh *static_meshes, int32_t n_static, const GxMesh *dyn_meshes, int32_t n_dyn,
                    int32_t cuda_device, GxScene **out) {
    if (!out) return fail(GX_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!static_meshes || n_static <= 0) return fail(GX_ERR_INVALID_ARG, "need at least one static mesh");
    if (n_dyn < 0 || (n_dyn > 0 && !dyn_meshes)) return fail(GX_ERR_INVALID_ARG, "bad dynamic mesh array");
    std::vector<float4> verts;
    std::vector<uchar4> tris;
    std::vector<GxBatchDev> batches;
    std::vector<GxClusterDev> clusters, subs;
    std::vector<GxMeshDev> meshes;
    GxScene *sc = new (std::nothrow) GxScene();
    if (!sc) return fail(GX_ERR_OOM, "host allocation failed");
    try {
        for (int i = 0; i < n_static + n_dyn; ++i) {
            const GxMesh &m = i < n_static ? static_meshes[i] : dyn_meshes[i - n_static];
            if ((m.nv && (!m.positions || !m.colors)) || (m.nt && !m.indices)) {
                delete sc;
                return fail(GX_ERR_INVALID_ARG, "mesh %d has NULL arrays", i);
            }
            GxMeshDev md;
            const size_t b0 = batches.size();
            const int rc = build_mesh(m, verts, tris, batches, subs, clusters, md);
            if (rc != GX_OK) { delete sc; return rc; }
            uint32_t &mb = i < n_static ? sc->max_static_batches : sc->max_dyn_batches;
            mb = std::max<uint32_t>(mb, (uint32_t)(batches.size() - b0));
            meshes.push_back(md);
            sc->mesh_nt.push_back(m.nt);
            if (i < n_static) sc->max_static_nt = std::max(sc->max_static_nt, m.nt);
            else sc->max_dyn_nt = std::max(sc->max_dyn_nt, m.nt);
        }
    } catch (const std::bad_alloc &) {
        delete sc;
        return fail(GX_ERR_OOM, "host allocation failed while clustering");
    }
    if (batches.size() >= (1u << 24) || verts.size() >= 0xFFFFFFFFull || tris.size() >= 0xFFFFFFFFull) {
        delete sc;
        return fail(GX_ERR_UNSUPPORTED, "scene too large: %zu batches", batches.size());
    }
    sc->device = cuda_device;
    sc->n_static = n_static;
    sc->n_dyn = n_dyn;
    DeviceGuard guard(cuda_device);
    int rc = GX_OK;
    if (!guard.ok) rc = fail(GX_ERR_CUDA, "cannot select CUDA device %d", cuda_device);
    cudaDeviceProp prop;
    if (rc == GX_OK && cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess)
        rc = fail(GX_ERR_CUDA, "cudaGetDeviceProperties failed");
    if (rc == GX_OK) {
        sc->num_sms = prop.multiProcessorCount;
        sc->max_smem_optin = (int)prop.sharedMemPerBlockOptin;
        for (const GxClusterDev &c : clusters) sc->max_nbatch = std::max(sc->max_nbatch, c.nbatch);
    }
    if (rc == GX_OK) rc = upload(sc->verts, verts);
    if (rc == GX_OK) rc = upload(sc->tris, tris);
    if (rc == GX_OK) rc = upload(sc->batches, batches);
    if (rc == GX_OK) rc = upload(sc->subs, subs);
    if (rc == GX_OK) rc = upload(sc->clusters, clusters);
    if (rc == GX_OK) rc = upload(sc->meshes, meshes);
    if (rc == GX_OK) {
        auto alloc = [&]() -> int {
            GX_CUDA(cudaMalloc(&sc->env_counter, sizeof(unsigned int)));
            GX_CUDA(cudaMalloc(&sc->stats, GX_NSTAT * sizeof(unsigned long long)));
            GX_CUDA(cudaMemset(sc->stats, 0, GX_NSTAT * sizeof(unsigned long long)));
            return GX_OK;
        };
        rc = alloc();
    }
    if (rc != GX_OK) {
        std::string keep = g_err;
        gx_destroy(sc);
        snprintf(g_err, sizeof(g_err), "%s", keep.c_str());
        return rc;
    }
    *out = sc;
    return GX_OK;
}

void gx_destroy(GxScene *sc) {
    if (!sc) return;
    DeviceGuard guard(sc->device);
    cudaFree(sc->verts);
    cudaFree(sc->tris);
    cudaFree(sc->batches);
    cudaFree(sc->subs);
    cudaFree(sc->clusters);
    cudaFree(sc->meshes);
    cudaFree(sc->env_counter);
    cudaFree(sc->stats);
    sc->pool.release(); sc->pipe_scratch.release(); sc->frames.release();
    for (cudaEvent_t e : sc->t_ev) cudaEventDestroy(e);
    if (sc->d_maxrec) cudaFree(sc->d_maxrec);
    if (sc->h_maxrec) cudaFreeHost(sc->h_maxrec);
    if (sc->ev_maxrec) cudaEventDestroy(sc->ev_maxrec);
    sc->h_env_scene.release(); sc->h_inst_mesh.release(); sc->h_cam_pose.release(); sc->h_inst_xform.release();
    sc->h_depth.release(); sc->h_rgb.release(); sc->h_id.release();
    if (sc->host_stream) cudaStreamDestroy(sc->host_stream);
    if (sc->copy_stream) cudaStreamDestroy(sc->copy_stream);
    if (sc->ev_sub) cudaEventDestroy(sc->ev_sub);
    delete sc;
}

int gx_set_option(GxScene *sc, const char *name, int64_t value) {
    if (!sc || !name) return fail(GX_ERR_INVALID_ARG, "NULL argument");
    if (!strcmp(name, "cull")) { sc->opt_cull = value != 0; return GX_OK; }
    if (!strcmp(name, "stats")) { sc->opt_stats = value != 0; return GX_OK; }
    if (!strcmp(name, "timing")) {   // 1 = start (and reset) the per-kernel event timing, 0 = stop recording
        sc->opt_timing = value != 0;
        if (value) { sc->t_used = 0; sc->t_calls = 0; }
        return GX_OK;
    }
    if (!strcmp(name, "subcull")) { sc->opt_subcull = value != 0; return GX_OK; }
    if (!strcmp(name, "bands")) {
        if (value != 0 && value != 1 && value != 2 && value != 4) return fail(GX_ERR_INVALID_ARG, "bands must be 0, 1, 2 or 4");
        sc->opt_bands = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "occlusion")) {
        if (value < 0 || value > 3) return fail(GX_ERR_INVALID_ARG, "occlusion must be 0 (off), 1 (automatic), 2 or 3 (passes)");
        sc->opt_occlusion = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "occl_area")) {
        if (value < 0 || value > 16384) return fail(GX_ERR_INVALID_ARG, "occl_area out of range");
        sc->opt_occl_area = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "occluder_pct")) {
        if (value < 1 || value > 100) return fail(GX_ERR_INVALID_ARG, "occluder_pct must be in [1, 100]");
        sc->opt_occluder_pct = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "path")) {
        if (value < 0 || value > 1) return fail(GX_ERR_INVALID_ARG, "path must be 0 or 1");
        sc->opt_path = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "pool_slots")) {
        if (value < 0 || value > (1 << 24)) return fail(GX_ERR_INVALID_ARG, "pool_slots out of range");
        sc->opt_pool_slots = value;
        return GX_OK;
    }
    if (!strcmp(name, "pool_bytes")) {
        if (value < 0) return fail(GX_ERR_INVALID_ARG, "pool_bytes must be >= 0");
        sc->opt_pool_bytes = value;
        return GX_OK;
    }
    if (!strcmp(name, "big_slots") || !strcmp(name, "chunk_slots")) {
        if (value < 32 || value > (1 << 20)) return fail(GX_ERR_INVALID_ARG, "%s must be in [32, 2^20]", name);
        (name[0] == 'b' ? sc->opt_big_slots : sc->opt_chunk_slots) = (int)value;
        return GX_OK;
    }
    return fail(GX_ERR_INVALID_ARG, "unknown option '%s'", name);
}

int gx_get_stat(GxScene *sc, const char *name, int64_t *out) {
    if (!sc || !name || !out) return fail(GX_ERR_INVALID_ARG, "NULL argument");
    if (!strcmp(name, "launches")) { *out = sc->last_launches; return GX_OK; }
    if (!strcmp(name, "timed_calls")) { *out = sc->t_calls; return GX_OK; }
    if (!strncmp(name, "ns_", 3)) {   // nanoseconds per kernel class, summed over the calls since "timing" was set
        static const char *kinds[6] = {"", "cull", "geom", "order", "raster", "fallback"};
        int kind = 0;
        for (int k = 1; k < 6; ++k) if (!strcmp(name + 3, kinds[k])) kind = k;
        if (!kind) return fail(GX_ERR_INVALID_ARG, "unknown stat '%s'", name);
        DeviceGuard guard(sc->device);
        if (sc->t_used) GX_CUDA(cudaEventSynchronize(sc->t_ev[sc->t_used - 1]));
        double ns = 0.0;
        for (size_t k = 1; k < sc->t_used; ++k)
            if (sc->t_kind[k] == kind) {
                float ms = 0.0f;
                GX_CUDA(cudaEventElapsedTime(&ms, sc->t_ev[k - 1], sc->t_ev[k]));
                ns += 1e6 * (double)ms;
            }
        *out = (int64_t)ns;
        return GX_OK;
    }
    if (!strcmp(name, "max_env_records") || !strcmp(name, "p50_env_records")) {   // last chunk of the two-kernel path
        *out = 0;
        if (sc->last_chunk_n <= 0) return GX_OK;
        DeviceGuard guard(sc->device);
        std::vector<uint32_t> cnt(2 * (size_t)sc->last_chunk_n);
        GX_CUDA(cudaStreamSynchronize(sc->last_stream));
        GX_CUDA(cudaMemcpy(cnt.data(), sc->pipe_scratch.p + 12, cnt.size() * 4, cudaMemcpyDeviceToHost));
        std::vector<uint32_t> tot(sc->last_chunk_n);
        for (int e = 0; e < sc->last_chunk_n; ++e) tot[e] = cnt[2 * e] + cnt[2 * e + 1];
        std::sort(tot.begin(), tot.end());
        *out = name[0] == 'm' ? tot.back() : tot[tot.size() / 2];
        return GX_OK;
    }
    static const char *names[GX_NSTAT] = {"clusters_tested", "clusters_drawn", "triangles_in", "triangles_raster",
                                          "fragments", "overflow_envs", "clusters_occluded", "records_occluded"};
    for (int k = 0; k < GX_NSTAT; ++k)
        if (!strcmp(name, names[k])) {
            DeviceGuard guard(sc->device);
            unsigned long long v[GX_NSTAT];
            GX_CUDA(cudaStreamSynchronize(sc->last_stream));
            GX_CUDA(cudaMemcpy(v, sc->stats, sizeof(v), cudaMemcpyDeviceToHost));
            *out = (int64_t)v[k];
            return GX_OK;
        }
    return fail(GX_ERR_INVALID_ARG, "unknown stat '%s'", name);
}

static int render_impl(GxScene *sc, const GxCamera *cam, int32_t N, int32_t K, const int32_t *env_scene,
                       const float *cam_pose, const int32_t *inst_mesh, const float *inst_xform, uint8_t *rgb_out,
                       float *depth_out, uint32_t *id_out, uint16_t *obs_out, float obs_dmin, float obs_dmax,
                       void *cuda_stream) {
    if (!sc || !cam) return fail(GX_ERR_INVALID_ARG, "NULL scene or camera");
    if (N <= 0) return fail(GX_ERR_INVALID_ARG, "N must be positive, got %d", N);
    if (K < 0 || K > GX_MAX_INSTANCES) return fail(GX_ERR_INVALID_ARG, "K must be in [0, %d], got %d", GX_MAX_INSTANCES, K);
    if (!env_scene || !cam_pose || (!depth_out && !obs_out))
        return fail(GX_ERR_INVALID_ARG, "env_scene, cam_pose and depth_out (or obs_out) are required");
    if (obs_out && !(obs_dmax > obs_dmin)) return fail(GX_ERR_INVALID_ARG, "need depth_min < depth_max");
    if (K > 0 && (!inst_mesh || !inst_xform)) return fail(GX_ERR_INVALID_ARG, "inst_mesh and inst_xform are required when K > 0");
    if (cam->width <= 0 || cam->height <= 0 || cam->width % 16 || cam->height % 16)
        return fail(GX_ERR_INVALID_ARG, "width and height must be positive multiples of 16, got %dx%d", cam->width, cam->height);
    if (!(cam->znear > 0.0f) || !(cam->zfar > cam->znear)) return fail(GX_ERR_INVALID_ARG, "need 0 < znear < zfar");
    if (!(cam->fx > 0.0f) || !(cam->fy > 0.0f)) return fail(GX_ERR_INVALID_ARG, "fx and fy must be positive");
    if ((long long)cam->width * cam->height > 16384)
        return fail(GX_ERR_UNSUPPORTED, "width*height = %lld exceeds 16384 (the frame must fit shared memory)",
                    (long long)cam->width * cam->height);
    if ((unsigned long long)sc->max_static_nt + (unsigned long long)K * sc->max_dyn_nt >= (1ull << 31))
        return fail(GX_ERR_UNSUPPORTED, "more than 2^31 triangles per environment");
    DeviceGuard guard(sc->device);
    if (!guard.ok) return fail(GX_ERR_CUDA, "cannot select CUDA device %d", sc->device);
    cudaStream_t stream = (cudaStream_t)cuda_stream;

    if (cam->width > 128 || cam->height > 128)
        return fail(GX_ERR_UNSUPPORTED, "width and height must be <= 128 in this build, got %dx%d", cam->width, cam->height);
    GxParams P;
    P.verts = sc->verts; P.tris = sc->tris; P.batches = sc->batches; P.subs = sc->subs; P.clusters = sc->clusters; P.meshes = sc->meshes;
    P.n_static = sc->n_static; P.n_dyn = sc->n_dyn;
    P.N = N; P.K = K; P.W = cam->width; P.H = cam->height;
    P.fx = cam->fx; P.fy = cam->fy; P.znear = cam->znear; P.zfar = cam->zfar;
    P.env_scene = env_scene; P.cam_pose = cam_pose; P.inst_mesh = inst_mesh; P.inst_xform = inst_xform;
    P.rgb = rgb_out; P.depth = depth_out; P.id = id_out;
    P.obs = obs_out; P.obs_dmin = obs_dmin; P.obs_range = obs_dmax - obs_dmin;
    P.env_counter = sc->env_counter; P.stats = sc->stats;
    P.env_filter = nullptr;
    P.cull = sc->opt_cull;
    P.cull_chunk = gx::WORK_CAP / (int)sc->max_nbatch;

    GX_CUDA(cudaMemsetAsync(sc->stats, 0, GX_NSTAT * sizeof(unsigned long long), stream));
    const bool st = sc->opt_stats != 0;
    sc->last_stream = stream;
    sc->last_chunk_n = 0;
    if (sc->opt_path == 1) {
        GX_CUDA(cudaMemsetAsync(sc->env_counter, 0, sizeof(unsigned int), stream));
        const int rc = launch_single(sc, P, stream, st);
        if (rc != GX_OK) return rc;
        sc->last_launches = 1;
        return GX_OK;
    }

    // ---- two-kernel path, in chunks of environments that share the record pool ----------------------
    const int64_t npix = (int64_t)P.W * P.H;
    // bands: (environment, band) is the raster task; several bands only if each is a multiple of 32 rows
    int bands = sc->opt_bands > 0 ? sc->opt_bands : (npix * 8 > 65536 ? 2 : 1);
    while (bands > 1 && (P.H % bands || (P.H / bands) % 32)) bands >>= 1;
    const int bh = P.H / bands;
    // pool segment per raster task: a default from the frame size, raised to 1.25 x the largest record count any
    // task of an earlier call on this handle produced (read back asynchronously; a call whose segments are too
    // small is still rendered correctly, by the overflow pass, and the next call is sized for it)
    if (!sc->d_maxrec) {
        GX_CUDA(cudaMalloc(&sc->d_maxrec, 2 * sizeof(uint32_t)));
        GX_CUDA(cudaMallocHost(&sc->h_maxrec, 2 * sizeof(uint32_t)));
        GX_CUDA(cudaEventCreateWithFlags(&sc->ev_maxrec, cudaEventDisableTiming));
    }
    if (sc->maxrec_pending && cudaEventQuery(sc->ev_maxrec) == cudaSuccess) {
        sc->hist_n = std::max(sc->hist_n, sc->h_maxrec[0]);
        sc->hist_w = std::max(sc->hist_w, sc->h_maxrec[1]);
        sc->maxrec_pending = false;
    }
    cudaGetLastError();   // (cudaErrorNotReady of the query is not an error)
    auto grow = [](uint32_t seen) { return ((int64_t)seen + seen / 4 + 1023) & ~(int64_t)1023; };
    const int64_t cap_n = sc->opt_pool_slots > 0 ? sc->opt_pool_slots
                                                 : std::max<int64_t>(std::max<int64_t>(2048, 4 * npix / bands), grow(sc->hist_n));
    const int64_t cap_w = sc->opt_pool_slots > 0 ? (std::max<int64_t>(64, cap_n / 8) & ~(int64_t)1)
                                                 : std::max<int64_t>(std::max<int64_t>(64, cap_n / 8) & ~(int64_t)1, grow(sc->hist_w));
    const int64_t env_bytes = (cap_n + cap_w) * 64 * bands;
    const int64_t budget = sc->opt_pool_bytes > 0 ? sc->opt_pool_bytes : (int64_t)8 << 30;
    const int chunk = (int)std::max<int64_t>(1, std::min<int64_t>(N, budget / env_bytes));
    int rc;
    if ((rc = sc->pool.reserve((size_t)chunk * bands * (size_t)(cap_n + cap_w) * 4)) != GX_OK) return rc;
    // scratch words: counters[12] | cnt[2*tasks] | env_flag[chunk] (zeroed per chunk) | order[tasks] | cnt1[2*tasks] |
    //                thr[chunk] | env_idb[chunk*(K+1)] | env_mv[chunk*(K+1)*12] | hiz[chunk*HZ_STRIDE] | items[4*...]
    // occluder scheme: 2 or 3 passes; automatic = 2 passes where they pay: frames of 8192 pixels or more (the hi-Z
    // tiles are 8x8 pixels) and enough environments that two rounds of kernels still fill the GPU
    const int n_pass = sc->opt_occlusion == 1 ? ((npix >= 8192 && N >= 512) ? 2 : 0) : sc->opt_occlusion;
    const bool two_phase = sc->opt_cull && n_pass >= 2;
    const size_t k1 = (size_t)K + 1, tasks = (size_t)chunk * bands;
    const size_t items_per_env = (size_t)sc->max_static_batches + (size_t)K * sc->max_dyn_batches;
    const size_t n_zero = 12 + 2 * tasks + (size_t)chunk;
    const size_t off_order = n_zero, off_cnt1 = off_order + tasks, off_thr = off_cnt1 + 2 * tasks;
    const size_t off_idb = off_thr + chunk, off_mv = off_idb + chunk * k1, off_hiz = off_mv + chunk * k1 * 12;
    const size_t off_items = (off_hiz + (size_t)chunk * gx::HZ_STRIDE + 3) & ~(size_t)3;
    if ((rc = sc->pipe_scratch.reserve(off_items + 4 * (size_t)chunk * std::max<size_t>(items_per_env, 1))) != GX_OK) return rc;
    if (two_phase && (rc = sc->frames.reserve((size_t)chunk * (size_t)npix)) != GX_OK) return rc;
    int launches = 0;
    GX_CUDA(cudaMemsetAsync(sc->d_maxrec, 0, 2 * sizeof(uint32_t), stream));
    for (int e0 = 0; e0 < N; e0 += chunk) {
        const int n = std::min(chunk, N - e0);
        gx::PipeParams PP;
        PP.g = P;
        PP.g.N = n;
        PP.g.env_scene = env_scene + e0;
        PP.g.cam_pose = cam_pose + (size_t)e0 * 16;
        PP.g.inst_mesh = inst_mesh ? inst_mesh + (size_t)e0 * K : nullptr;
        PP.g.inst_xform = inst_xform ? inst_xform + (size_t)e0 * K * 16 : nullptr;
        PP.g.rgb = rgb_out ? rgb_out + (size_t)e0 * npix * 3 : nullptr;
        PP.g.depth = depth_out ? depth_out + (size_t)e0 * npix : nullptr;
        PP.g.obs = obs_out ? obs_out + (size_t)e0 * npix * 4 : nullptr;
        PP.g.id = id_out ? id_out + (size_t)e0 * npix : nullptr;
        PP.recs = sc->pool.p;
        PP.counters = sc->pipe_scratch.p;
        PP.cnt = sc->pipe_scratch.p + 12;
        PP.env_flag = sc->pipe_scratch.p + 12 + 2 * tasks;
        PP.cnt1 = sc->pipe_scratch.p + off_cnt1;
        PP.thr = reinterpret_cast<float *>(sc->pipe_scratch.p + off_thr);
        PP.hiz = reinterpret_cast<float *>(sc->pipe_scratch.p + off_hiz);
        PP.frames = sc->frames.p;
        PP.occl_pct = two_phase ? sc->opt_occluder_pct : 100;
        PP.cap_n = (int32_t)cap_n;
        PP.cap_w = (int32_t)cap_w;
        PP.bands = bands;
        PP.subcull = sc->opt_cull && sc->opt_subcull;
        PP.phase = 0;
        PP.bh = bh;
        PP.big_slots = sc->opt_big_slots;
        PP.chunk_slots = sc->opt_chunk_slots;
        PP.order = sc->pipe_scratch.p + off_order;
        PP.maxrec = sc->d_maxrec;
        PP.env_idb = sc->pipe_scratch.p + off_idb;
        PP.env_mv = reinterpret_cast<float *>(sc->pipe_scratch.p + off_mv);
        PP.items = reinterpret_cast<uint4 *>(sc->pipe_scratch.p + off_items);
        GX_CUDA(cudaMemsetAsync(sc->pipe_scratch.p, 0, n_zero * sizeof(uint32_t), stream));
        PP.nphase = two_phase ? n_pass : 0;
        PP.occl_area = (float)sc->opt_occl_area;
        if (!two_phase) {
            if ((rc = launch_pass<0>(sc, PP, stream, st)) != GX_OK) return rc;
            launches += 4;
        } else {
            PP.phase = 1;
            if ((rc = launch_pass<1>(sc, PP, stream, st)) != GX_OK) return rc;
            if (PP.nphase == 3) {
                PP.counters = sc->pipe_scratch.p + 8;
                PP.phase = 2;
                if ((rc = launch_pass<3>(sc, PP, stream, st)) != GX_OK) return rc;
                launches += 4;
            }
            PP.counters = sc->pipe_scratch.p + 4;
            PP.phase = PP.nphase;
            if ((rc = launch_pass<2>(sc, PP, stream, st)) != GX_OK) return rc;
            launches += 8;
        }
        // environments whose records overflowed their pool segment: single-kernel pass over the flagged ones
        GxParams PL = PP.g;
        PL.env_counter = sc->pipe_scratch.p + 3;
        PL.env_filter = PP.env_flag;
        if ((rc = launch_single(sc, PL, stream, st)) != GX_OK) return rc;
        if ((rc = mark(sc, stream, 5)) != GX_OK) return rc;
        launches += 1;
        sc->last_chunk_n = n * bands;
    }
    if (!sc->maxrec_pending) {   // (a read-back still in flight keeps its buffer)
        GX_CUDA(cudaMemcpyAsync(sc->h_maxrec, sc->d_maxrec, 2 * sizeof(uint32_t), cudaMemcpyDeviceToHost, stream));
        GX_CUDA(cudaEventRecord(sc->ev_maxrec, stream));
        sc->maxrec_pending = true;
    }
    sc->last_launches = launches;
    if (sc->opt_timing) ++sc->t_calls;
    return GX_OK;
}


int gx_render_batch(GxScene *sc, const GxCamera *cam, int32_t N, int32_t K, const int32_t *env_scene,
                    const float *cam_pose, const int32_t *inst_mesh, const float *inst_xform, uint8_t *rgb_out,
                    float *depth_out, uint32_t *id_out, void *cuda_stream) {
    if (!depth_out) return fail(GX_ERR_INVALID_ARG, "depth_out is required");
    return render_impl(sc, cam, N, K, env_scene, cam_pose, inst_mesh, inst_xform, rgb_out, depth_out, id_out, nullptr, 0.0f,
                       1.0f, cuda_stream);
}

int gx_render_batch_obs(GxScene *sc, const GxCamera *cam, int32_t N, int32_t K, const int32_t *env_scene,
                        const float *cam_pose, const int32_t *inst_mesh, const float *inst_xform, uint16_t *obs_out,
                        float depth_min, float depth_max, void *cuda_stream) {
    if (!obs_out) return fail(GX_ERR_INVALID_ARG, "obs_out is required");
    return render_impl(sc, cam, N, K, env_scene, cam_pose, inst_mesh, inst_xform, nullptr, nullptr, nullptr, obs_out, depth_min,
                       depth_max, cuda_stream);
}

int gx_render_batch_host(GxScene *sc, const GxCamera *cam, int32_t N, int32_t K, const int32_t *env_scene,
                         const float *cam_pose, const int32_t *inst_mesh, const float *inst_xform, uint8_t *rgb_out,
                         float *depth_out, uint32_t *id_out) {
    if (!sc || !cam) return fail(GX_ERR_INVALID_ARG, "NULL scene or camera");
    if (N <= 0 || K < 0) return fail(GX_ERR_INVALID_ARG, "bad N or K");
    if (!env_scene || !cam_pose || !depth_out || (K > 0 && (!inst_mesh || !inst_xform)))
        return fail(GX_ERR_INVALID_ARG, "NULL array argument");
    if (cam->width <= 0 || cam->height <= 0) return fail(GX_ERR_INVALID_ARG, "bad camera size");
    DeviceGuard guard(sc->device);
    if (!guard.ok) return fail(GX_ERR_CUDA, "cannot select CUDA device %d", sc->device);
    if (!sc->host_stream) GX_CUDA(cudaStreamCreateWithFlags(&sc->host_stream, cudaStreamNonBlocking));
    cudaStream_t st = sc->host_stream;
    const size_t npix = (size_t)cam->width * cam->height, nk = (size_t)N * K;
    int rc;
    if ((rc = sc->h_env_scene.reserve(N)) || (rc = sc->h_cam_pose.reserve((size_t)N * 16)) ||
        (rc = sc->h_inst_mesh.reserve(std::max<size_t>(nk, 1))) || (rc = sc->h_inst_xform.reserve(std::max<size_t>(nk * 16, 1))) ||
        (rc = sc->h_depth.reserve(N * npix)) || (rgb_out && (rc = sc->h_rgb.reserve(N * npix * 3))) ||
        (id_out && (rc = sc->h_id.reserve(N * npix))))
        return rc;
    GX_CUDA(cudaMemcpyAsync(sc->h_env_scene.p, env_scene, (size_t)N * 4, cudaMemcpyHostToDevice, st));
    GX_CUDA(cudaMemcpyAsync(sc->h_cam_pose.p, cam_pose, (size_t)N * 64, cudaMemcpyHostToDevice, st));
    if (K > 0) {
        GX_CUDA(cudaMemcpyAsync(sc->h_inst_mesh.p, inst_mesh, nk * 4, cudaMemcpyHostToDevice, st));
        GX_CUDA(cudaMemcpyAsync(sc->h_inst_xform.p, inst_xform, nk * 64, cudaMemcpyHostToDevice, st));
    }
    // render in sub-batches of 512 environments and copy each one's images back on a second stream while the next
    // one renders (the device-to-host copy of RGBD is as long as the rendering itself)
    if (!sc->copy_stream) {
        GX_CUDA(cudaStreamCreateWithFlags(&sc->copy_stream, cudaStreamNonBlocking));
        GX_CUDA(cudaEventCreateWithFlags(&sc->ev_sub, cudaEventDisableTiming));
    }
    const int sub = 512;
    for (int e0 = 0; e0 < N; e0 += sub) {
        const int n = std::min(sub, N - e0);
        const size_t o = (size_t)e0 * npix, cnt = (size_t)n * npix;
        rc = gx_render_batch(sc, cam, n, K, sc->h_env_scene.p + e0, sc->h_cam_pose.p + (size_t)e0 * 16,
                             K > 0 ? sc->h_inst_mesh.p + (size_t)e0 * K : nullptr,
                             K > 0 ? sc->h_inst_xform.p + (size_t)e0 * K * 16 : nullptr,
                             rgb_out ? sc->h_rgb.p + o * 3 : nullptr, sc->h_depth.p + o, id_out ? sc->h_id.p + o : nullptr, st);
        if (rc != GX_OK) return rc;
        GX_CUDA(cudaEventRecord(sc->ev_sub, st));
        GX_CUDA(cudaStreamWaitEvent(sc->copy_stream, sc->ev_sub, 0));
        GX_CUDA(cudaMemcpyAsync(depth_out + o, sc->h_depth.p + o, cnt * 4, cudaMemcpyDeviceToHost, sc->copy_stream));
        if (rgb_out) GX_CUDA(cudaMemcpyAsync(rgb_out + o * 3, sc->h_rgb.p + o * 3, cnt * 3, cudaMemcpyDeviceToHost, sc->copy_stream));
        if (id_out) GX_CUDA(cudaMemcpyAsync(id_out + o, sc->h_id.p + o, cnt * 4, cudaMemcpyDeviceToHost, sc->copy_stream));
    }
    GX_CUDA(cudaStreamSynchronize(sc->copy_stream));
    GX_CUDA(cudaStreamSynchronize(st));
    return GX_OK;
}

}  // extern "C"
