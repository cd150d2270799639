// gx_api.cu -- host side of the C ABI declared in include/gx.h: scene upload (clustering), launch, errors.
// Product code.  Nothing here includes, links or calls anything under oracle/.
#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/gx.h"
#include "gx_pipeline.cuh"
#include "gx_fk.cuh"
#include "gx_collide.cuh"

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
    bool in_graph = false;   // a captured CUDA graph holds this buffer's address
    // grow only; contents are not kept.  A buffer a graph may still use is not freed but handed to `retired`
    // (gx_destroy frees that list), so that replaying the graph stays valid
    int reserve(size_t want, std::vector<void *> *retired = nullptr) {
        if (want <= n) return GX_OK;
        if (p && in_graph && retired) {
            try { retired->push_back(p); } catch (const std::bad_alloc &) { return fail(GX_ERR_OOM, "host allocation failed"); }
        } else if (p) cudaFree(p);
        p = nullptr;
        n = 0;
        in_graph = false;
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
    uint32_t max_dyn_nt = 0, max_static_nt = 0;
    uint32_t max_static_batches = 0, max_dyn_batches = 0;   // largest number of batches in any static / dynamic mesh
    int max_smem_optin = 0;
    int64_t default_pool_bytes = (int64_t)4 << 30;   // arena budget: set by gx_create_scene to an eighth of the device's memory, at most 16 GB
    unsigned long long *stats = nullptr;   // device [GX_NSTAT]
    // options (gx_set_option)
    int opt_cull = 1, opt_subcull = 1, opt_stats = 0, opt_hiz = 1, opt_big_px = 24;
    int opt_bin_threads = 0;
    int opt_max_rounds = 0;             // rounds of stage kernels the host launches at most (0 = no limit; 1 = later waves all in the tail kernel)
    int opt_ctas_per_sm = 0;            // persistent kernels: CTAs per SM (0 = as many as fit); smaller when two handles share the GPU
    int opt_host_sub = 0;               // gx_render_batch_host: environments per sub-batch; 0 = automatic
    int opt_occlusion = -1;             // occluder scheme: 1 on, 0 off, -1 automatic (on for frames of at least 4096 pixels)
    int opt_occl_area = 64;             // pixels per triangle of a sub-cluster's screen box that make it an occluder
    int64_t opt_pool_bytes = 0;         // arena budget; 0 = default_pool_bytes (an eighth of the device's memory, at most 16 GB)
    int64_t opt_arena_slots = 0;        // force the arena size in record slots (tests: several waves); 0 = automatic
    // scratch owned by the handle: grows on demand, never inside a steady-state call
    DevBuf<uint4> arena_recs;
    DevBuf<uint2> arena_bbs;
    DevBuf<uint32_t> arena_refs;
    size_t arena_slots = 0;
    DevBuf<uint32_t> scratch;           // ctl | per-environment tables | tile offsets | task lists | items
    // arena sizing from history: the per-environment mean and the maximum of U of earlier calls
    uint32_t *h_ctl = nullptr;          // pinned host copy of the control words of the last call
    cudaEvent_t ev_ctl = nullptr;
    bool ctl_pending = false;
    bool capturing = false;             // the current call's stream is being captured into a CUDA graph
    std::vector<void *> retired;        // buffers a captured graph may still use, replaced by larger ones since; freed by gx_destroy
    int ctl_N = 0;
    double hist_u_per_env = 0.0;
    int hist_waves = 1;                 // waves the last call needed (the host launches that many rounds of the stage kernels)
    // kernel timing (option "timing"): CUDA events recorded on the caller's stream around every kernel
    int opt_timing = 0;
    std::vector<cudaEvent_t> t_ev;      // recorded marks, in order
    std::vector<int> t_kind;            // what ran before the mark: 0 = start of a call, 1 cull, 2 geom, 3 bin, 4 raster, 5 tail
    size_t t_used = 0;
    int t_calls = 0;
    bool t_full = false;
    int last_launches = 0;
    cudaStream_t last_stream = nullptr;
    // launch configurations, resolved once per kernel instantiation (occupancy queries are not free)
    struct Plan { const void *fn; size_t smem; int threads; int per_sm; };
    std::vector<Plan> plans;
    // robot description (gx_set_robot)
    gx::FkLink *fk_links = nullptr;
    int fk_L = 0, fk_camera_link = -1, fk_ee_link = -1;
    float fk_mount[12] = {1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0};
    // collision world (gx_set_collision_world)
    float4 *mesh_box = nullptr;          // [n_dyn][2] object-space box of every dynamic mesh (centre, half extent)
    gx::ColGridDev *cg_grids = nullptr;
    uint32_t *cg_col_off = nullptr;
    float2 *cg_layers = nullptr;
    float *cg_radii = nullptr;
    gx::SphereDev *cg_spheres = nullptr;
    int cg_n_radii = 0, cg_S = 0, cg_max_link = -1;
    // staging for gx_render_batch_host
    DevBuf<int32_t> h_env_scene, h_inst_mesh;
    DevBuf<float> h_cam_pose, h_inst_xform, h_depth;
    DevBuf<uint8_t> h_rgb;
    DevBuf<uint32_t> h_id;
    cudaStream_t host_stream = nullptr, copy_stream = nullptr;
    std::vector<cudaEvent_t> ev_sub;
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

// blocks per SM of a kernel at a block size and dynamic shared memory size; sets the opt-in attribute once
int plan_of(GxScene *sc, const void *fn, int threads, size_t smem, int *per_sm) {
    for (const GxScene::Plan &p : sc->plans)
        if (p.fn == fn && p.smem == smem && p.threads == threads) { *per_sm = p.per_sm; return GX_OK; }
    GX_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int n = 0;
    GX_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, fn, threads, smem));
    if (n < 1) return fail(GX_ERR_UNSUPPORTED, "kernel does not fit: %zu bytes of shared memory", smem);
    sc->plans.push_back({fn, smem, threads, n});
    *per_sm = n;
    return GX_OK;
}

// timing mark: an event on the stream; the time since the previous mark belongs to kernel class `kind`
int mark(GxScene *sc, cudaStream_t stream, int kind) {
    if (!sc->opt_timing || sc->t_full) return GX_OK;
    if (sc->t_used >= 8192) { sc->t_full = true; return GX_OK; }
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
        sc->default_pool_bytes = std::min<int64_t>((int64_t)16 << 30, (int64_t)(prop.totalGlobalMem / 8));
    }
    if (rc == GX_OK) rc = upload(sc->verts, verts);
    if (rc == GX_OK) rc = upload(sc->tris, tris);
    if (rc == GX_OK) rc = upload(sc->batches, batches);
    if (rc == GX_OK) rc = upload(sc->subs, subs);
    if (rc == GX_OK) rc = upload(sc->clusters, clusters);
    if (rc == GX_OK) rc = upload(sc->meshes, meshes);
    if (rc == GX_OK) {   // N13: object-space box of every dynamic mesh, in binary32 as the definition says
        std::vector<float4> boxes((size_t)std::max(n_dyn, 1) * 2, make_float4(0.f, 0.f, 0.f, 0.f));
        for (int i = 0; i < n_dyn; ++i) {
            const GxMesh &m = dyn_meshes[i];
            float lo[3] = {0.f, 0.f, 0.f}, hi[3] = {0.f, 0.f, 0.f};
            for (uint32_t v = 0; v < m.nv; ++v)
                for (int a = 0; a < 3; ++a) {
                    const float pv = m.positions[3 * (size_t)v + a];
                    if (v == 0 || pv < lo[a]) lo[a] = pv;
                    if (v == 0 || pv > hi[a]) hi[a] = pv;
                }
            float c[3], h[3];
            for (int a = 0; a < 3; ++a) {
                volatile float sum = lo[a] + hi[a], dif = hi[a] - lo[a];   // (binary32 results, whatever the host compiler keeps in registers)
                c[a] = 0.5f * sum;
                h[a] = 0.5f * dif;
            }
            boxes[2 * (size_t)i] = make_float4(c[0], c[1], c[2], 0.f);
            boxes[2 * (size_t)i + 1] = make_float4(h[0], h[1], h[2], 0.f);
        }
        rc = upload(sc->mesh_box, boxes);
    }
    if (rc == GX_OK) {
        auto alloc = [&]() -> int {
            GX_CUDA(cudaMalloc(&sc->stats, GX_NSTAT * sizeof(unsigned long long)));
            GX_CUDA(cudaMemset(sc->stats, 0, GX_NSTAT * sizeof(unsigned long long)));
            GX_CUDA(cudaMallocHost(&sc->h_ctl, gx::C_NCTL * sizeof(uint32_t)));
            memset(sc->h_ctl, 0, gx::C_NCTL * sizeof(uint32_t));
            GX_CUDA(cudaEventCreateWithFlags(&sc->ev_ctl, cudaEventDisableTiming));
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
    cudaFree(sc->stats);
    cudaFree(sc->fk_links);
    cudaFree(sc->mesh_box); cudaFree(sc->cg_grids); cudaFree(sc->cg_col_off); cudaFree(sc->cg_layers); cudaFree(sc->cg_radii);
    cudaFree(sc->cg_spheres);
    sc->arena_recs.release(); sc->arena_bbs.release(); sc->arena_refs.release(); sc->scratch.release();
    for (void *q : sc->retired) cudaFree(q);
    for (cudaEvent_t e : sc->t_ev) cudaEventDestroy(e);
    if (sc->h_ctl) cudaFreeHost(sc->h_ctl);
    if (sc->ev_ctl) cudaEventDestroy(sc->ev_ctl);
    sc->h_env_scene.release(); sc->h_inst_mesh.release(); sc->h_cam_pose.release(); sc->h_inst_xform.release();
    sc->h_depth.release(); sc->h_rgb.release(); sc->h_id.release();
    if (sc->host_stream) cudaStreamDestroy(sc->host_stream);
    if (sc->copy_stream) cudaStreamDestroy(sc->copy_stream);
    for (cudaEvent_t e : sc->ev_sub) cudaEventDestroy(e);
    delete sc;
}

int gx_set_option(GxScene *sc, const char *name, int64_t value) {
    if (!sc || !name) return fail(GX_ERR_INVALID_ARG, "NULL argument");
    if (!strcmp(name, "cull")) { sc->opt_cull = value != 0; return GX_OK; }
    if (!strcmp(name, "subcull")) { sc->opt_subcull = value != 0; return GX_OK; }
    if (!strcmp(name, "hiz")) { sc->opt_hiz = value != 0; return GX_OK; }
    if (!strcmp(name, "stats")) { sc->opt_stats = value != 0; return GX_OK; }
    if (!strcmp(name, "timing")) {   // 1 = start (and reset) the per-kernel event timing, 0 = stop recording
        sc->opt_timing = value != 0;
        if (value) { sc->t_used = 0; sc->t_calls = 0; sc->t_full = false; }
        return GX_OK;
    }
    if (!strcmp(name, "ctas_per_sm")) {
        if (value < 0 || value > 8) return fail(GX_ERR_INVALID_ARG, "ctas_per_sm must be in [0, 8]");
        sc->opt_ctas_per_sm = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "max_rounds")) {   // (development / tests)
        if (value < 0) return fail(GX_ERR_INVALID_ARG, "max_rounds must be >= 0");
        sc->opt_max_rounds = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "bin_threads")) {   // (development)
        if (value != 0 && value != 256 && value != 512) return fail(GX_ERR_INVALID_ARG, "bin_threads must be 0, 256 or 512");
        sc->opt_bin_threads = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "host_sub")) {
        if (value < 0) return fail(GX_ERR_INVALID_ARG, "host_sub must be >= 0");
        sc->opt_host_sub = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "occlusion")) {
        if (value < -1 || value > 1) return fail(GX_ERR_INVALID_ARG, "occlusion must be -1 (automatic), 0 or 1");
        sc->opt_occlusion = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "occl_area")) {
        if (value < 0 || value > (1 << 20)) return fail(GX_ERR_INVALID_ARG, "occl_area out of range");
        sc->opt_occl_area = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "big_px")) {
        if (value < 1 || value > 2 * gx::TILE) return fail(GX_ERR_INVALID_ARG, "big_px must be in [1, %d]", 2 * gx::TILE);   // (a box below 32 pixels touches at most 3x3 tiles)
        sc->opt_big_px = (int)value;
        return GX_OK;
    }
    if (!strcmp(name, "pool_bytes")) {
        if (value < 0) return fail(GX_ERR_INVALID_ARG, "pool_bytes must be >= 0");
        sc->opt_pool_bytes = value;
        return GX_OK;
    }
    if (!strcmp(name, "arena_slots")) {
        if (value < 0 || value > 0xFFFFFFFFll) return fail(GX_ERR_INVALID_ARG, "arena_slots out of range");
        sc->opt_arena_slots = value;
        return GX_OK;
    }
    return fail(GX_ERR_INVALID_ARG, "unknown option '%s'", name);
}

int gx_get_stat(GxScene *sc, const char *name, int64_t *out) {
    if (!sc || !name || !out) return fail(GX_ERR_INVALID_ARG, "NULL argument");
    if (!strcmp(name, "launches")) { *out = sc->last_launches; return GX_OK; }
    if (!strcmp(name, "timed_calls")) { *out = sc->t_calls; return GX_OK; }
    if (!strcmp(name, "arena_bytes")) { *out = (int64_t)(sc->arena_slots * 88); return GX_OK; }
    if (!strcmp(name, "scratch_bytes")) { *out = (int64_t)(sc->scratch.n * sizeof(uint32_t)); return GX_OK; }
    if (!strncmp(name, "ns_", 3)) {   // nanoseconds per kernel class, summed over the calls since "timing" was set
        static const char *kinds[6] = {"", "cull", "geom", "bin", "raster", "tail"};
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
    {   // control words of the most recent call: waves, the sum and maximum of the per-environment slot bounds
        static const char *cnames[4] = {"waves", "sum_slots", "max_env_slots", "bad_ids"};
        for (int k = 0; k < 4; ++k)
            if (!strcmp(name, cnames[k])) {
                DeviceGuard guard(sc->device);
                if (!sc->scratch.p) { *out = 0; return GX_OK; }
                uint32_t c[gx::C_NCTL];
                GX_CUDA(cudaStreamSynchronize(sc->last_stream));
                GX_CUDA(cudaMemcpy(c, sc->scratch.p, sizeof(c), cudaMemcpyDeviceToHost));
                if (k == 0) *out = c[gx::C_WAVES];
                else if (k == 1) *out = (int64_t)((uint64_t)c[gx::C_SUM_U] | ((uint64_t)c[gx::C_SUM_U + 1] << 32));
                else if (k == 2) *out = c[gx::C_MAX_U];
                else *out = c[gx::C_BAD_ENVS];
                return GX_OK;
            }
    }
    static const char *names[GX_NSTAT] = {"clusters_tested", "clusters_drawn", "triangles_in", "triangles_raster",
                                          "fragments", "records_occluded", "blocks_drawn", "tile_refs", "triangles_hidden",
                                          "subclusters_hidden", "large_records", "large_draws", "bound_violations"};
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

// Arena and scratch for a call of this shape: allocates (or grows) what the handle owns and fills the pointers of
// PP.  PP.g.{N,K,W,H}, PP.T, PP.tiles_x/y and PP.occl must be set.  Allocation happens only when something has to
// grow (it may synchronise the device); gx_reserve does it ahead of the first render call.
static int setup_buffers(GxScene *sc, gx::PipeParams &PP, unsigned long long worst_tris) {
    GxParams &P = PP.g;
    const int N = P.N, K = P.K;
    int rc;
    // ---- arena: record slots shared by the environments of a wave ------------------------------------
    // An environment's segment is sized by U, the bound cull_kernel computes; the arena must hold the largest
    // possible U (four slots per triangle: everything clipped by the near plane into two pieces with float
    // colours), so that a wave always has room for at least one environment.  Beyond that it is sized from the
    // history of earlier calls (mean U per environment, read back asynchronously) or, on the first call, from a
    // default of 48 Ki slots per environment, and capped by the budget; what does not fit goes to later waves.
    if (!sc->capturing && sc->ctl_pending && cudaEventQuery(sc->ev_ctl) == cudaSuccess) {
        const uint64_t sum = (uint64_t)sc->h_ctl[gx::C_SUM_U] | ((uint64_t)sc->h_ctl[gx::C_SUM_U + 1] << 32);
        sc->hist_u_per_env = std::max(sc->hist_u_per_env, (double)sum / (double)std::max(sc->ctl_N, 1));
        sc->hist_waves = (int)std::min<uint32_t>(std::max<uint32_t>(sc->h_ctl[gx::C_WAVES], 1u), 256u);
        sc->ctl_pending = false;
    }
    cudaGetLastError();   // (cudaErrorNotReady of the query is not an error)
    const uint64_t worst_env = 4ull * worst_tris + 64;
    const int64_t budget = sc->opt_pool_bytes > 0 ? sc->opt_pool_bytes : sc->default_pool_bytes;
    uint64_t want;
    if (sc->opt_arena_slots > 0) want = (uint64_t)sc->opt_arena_slots;
    else {
        const double per_env = sc->hist_u_per_env > 0.0 ? 1.25 * sc->hist_u_per_env + 1024.0 : (double)std::min<uint64_t>(worst_env, 49152);
        want = std::min<uint64_t>((uint64_t)(per_env * N), (uint64_t)N * worst_env);
        want = std::min<uint64_t>(want, (uint64_t)budget / 88);
    }
    want = std::min<uint64_t>(std::max<uint64_t>(want, worst_env), 0xFFFFFF00ull);
    if (want > sc->arena_slots && sc->capturing) want = sc->arena_slots;   // (no allocation inside a capture: more waves instead)
    if (sc->capturing && sc->arena_slots < worst_env)
        return fail(GX_ERR_UNSUPPORTED, "the arena cannot hold one environment of this shape: call gx_reserve (or render once) before capturing the call into a CUDA graph");
    // Buffers whose addresses a captured graph holds are never freed while the handle lives: when one has to grow it is
    // retired instead, so that replaying the earlier graph stays valid (it keeps the arena it was captured with).
    std::vector<void *> *keep = &sc->retired;
    if (want > sc->arena_slots) {
        // the three arrays grow one by one and any of the allocations can fail: until all of them have the new size the
        // handle holds no arena at all, so that a later (smaller) call allocates again instead of trusting a stale size
        sc->arena_slots = 0;
        if ((rc = sc->arena_recs.reserve((size_t)want * 4, keep)) != GX_OK) return rc;
        if ((rc = sc->arena_bbs.reserve((size_t)want, keep)) != GX_OK) return rc;
        if ((rc = sc->arena_refs.reserve((size_t)want * 4, keep)) != GX_OK) return rc;
        sc->arena_slots = (size_t)want;
    }
    PP.recs = sc->arena_recs.p; PP.bbs = sc->arena_bbs.p; PP.refs = sc->arena_refs.p;
    // (never more than is held: inside a capture the arena does not grow, whatever "arena_slots" asks for)
    PP.arena_slots = (uint32_t)std::min<uint64_t>(sc->opt_arena_slots > 0 ? std::max<uint64_t>((uint64_t)sc->opt_arena_slots, worst_env) : (uint64_t)sc->arena_slots,
                                                  (uint64_t)sc->arena_slots);

    // ---- scratch words: ctl | U | rec_base | cnt | cntA | n_large | env_idb | env_mv | tile_off | tasks | hizt | hizb | items | keys
    const size_t n = (size_t)N, k1 = (size_t)K + 1, NK1 = (size_t)PP.T * gx::NBUCKET + 1;
    PP.item_stride = (int32_t)std::max<size_t>((size_t)sc->max_static_batches + (size_t)K * sc->max_dyn_batches, 1);
    size_t off = 64;
    const size_t o_U = off; off += n;
    const size_t o_nitems = off; off += n;
    const size_t o_cpre = off; off += n + 1;
    const size_t o_base = off; off += n;
    const size_t o_cnt = off; off += n;
    const size_t o_cntA = off; off += n;
    const size_t o_nl = off; off += n;
    const size_t o_idb = off; off += n * k1;
    const size_t o_mv = off; off += n * k1 * 12;
    const size_t o_toff = off; off += n * NK1;
    const size_t o_tasks = off; off += (size_t)gx::NCLASS * n * (size_t)PP.T;
    PP.hz_stride = 0;
    for (int w = PP.tiles_x, h = PP.tiles_y;; w = (w + 1) >> 1, h = (h + 1) >> 1) { PP.hz_stride += w * h; if (w == 1 && h == 1) break; }
    const size_t o_hizt = off; off += PP.occl ? n * (size_t)PP.hz_stride : 0;
    const size_t o_hizb = off; off += PP.occl ? n * (size_t)PP.T * 8 : 0;
    off = (off + 3) & ~(size_t)3;
    const size_t o_items = off; off += 4 * n * (size_t)PP.item_stride;
    const size_t o_witems = off; off += 4 * n * (size_t)PP.item_stride;
    const size_t o_witems2 = off; off += PP.occl ? 4 * n * (size_t)PP.item_stride : 0;
    const size_t o_keys = off; off += PP.occl ? n * (size_t)P.W * (size_t)P.H * 2 : 0;
    if (off > sc->scratch.n && sc->capturing)
        return fail(GX_ERR_UNSUPPORTED, "the handle's tables would have to grow during stream capture: call gx_reserve for this shape first");
    if ((rc = sc->scratch.reserve(off, keep)) != GX_OK) return rc;
    if (sc->capturing)   // (what this call enqueues is recorded with these addresses)
        sc->arena_recs.in_graph = sc->arena_bbs.in_graph = sc->arena_refs.in_graph = sc->scratch.in_graph = true;
    uint32_t *sp = sc->scratch.p;
    PP.ctl = sp; PP.U = sp + o_U; PP.n_items = sp + o_nitems; PP.item_pre = sp + o_cpre; PP.rec_base = sp + o_base;
    PP.cnt = sp + o_cnt; PP.cntA = sp + o_cntA; PP.n_large = sp + o_nl; PP.env_idb = sp + o_idb;
    PP.env_mv = reinterpret_cast<float *>(sp + o_mv);
    PP.tile_off = sp + o_toff; PP.tasks = sp + o_tasks; PP.hizt = sp + o_hizt; PP.hizb = sp + o_hizb;
    PP.items = reinterpret_cast<uint4 *>(sp + o_items);
    PP.wave_items = reinterpret_cast<uint4 *>(sp + o_witems);
    PP.wave_items2 = reinterpret_cast<uint4 *>(sp + o_witems2);
    PP.keys = reinterpret_cast<unsigned long long *>(sp + o_keys);

    return GX_OK;
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
    if (cam->width > GX_MAX_FRAME || cam->height > GX_MAX_FRAME)
        return fail(GX_ERR_UNSUPPORTED, "width and height must be <= %d (8-bit box fields of a record), got %dx%d",
                    GX_MAX_FRAME, cam->width, cam->height);
    const unsigned long long worst_tris = (unsigned long long)sc->max_static_nt + (unsigned long long)K * sc->max_dyn_nt;
    if (worst_tris >= (1ull << 29)) return fail(GX_ERR_UNSUPPORTED, "more than 2^29 triangles per environment");
    if ((unsigned long long)N * (unsigned long long)((cam->width / 16) * (cam->height / 16)) >= (1ull << 31))
        return fail(GX_ERR_UNSUPPORTED, "more than 2^31 tiles per call");
    DeviceGuard guard(sc->device);
    if (!guard.ok) return fail(GX_ERR_CUDA, "cannot select CUDA device %d", sc->device);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const bool st = sc->opt_stats != 0;

    gx::PipeParams PP;
    GxParams &P = PP.g;
    P.verts = sc->verts; P.tris = sc->tris; P.batches = sc->batches; P.subs = sc->subs; P.clusters = sc->clusters; P.meshes = sc->meshes;
    P.n_static = sc->n_static; P.n_dyn = sc->n_dyn;
    P.N = N; P.K = K; P.W = cam->width; P.H = cam->height;
    P.fx = cam->fx; P.fy = cam->fy; P.znear = cam->znear; P.zfar = cam->zfar;
    P.env_scene = env_scene; P.cam_pose = cam_pose; P.inst_mesh = inst_mesh; P.inst_xform = inst_xform;
    P.rgb = rgb_out; P.depth = depth_out; P.id = id_out;
    P.obs = obs_out; P.obs_dmin = obs_dmin; P.obs_dmax = obs_dmax; P.obs_range = obs_dmax - obs_dmin;
    P.stats = sc->stats;
    P.cull = sc->opt_cull;
    PP.tiles_x = P.W / gx::TILE; PP.tiles_y = P.H / gx::TILE; PP.T = PP.tiles_x * PP.tiles_y;
    PP.bucket_off = -log2f(P.znear);
    PP.bucket_scale = (float)gx::NBUCKET / log2f(P.zfar / P.znear);
    PP.subcull = sc->opt_subcull;
    PP.big_px = sc->opt_big_px;
    PP.hiz = sc->opt_hiz;
    PP.occl = sc->opt_hiz && (sc->opt_occlusion == 1 || (sc->opt_occlusion < 0 && P.W * P.H >= 4096)) ? 1 : 0;
    PP.occl_area = (float)sc->opt_occl_area;

    int rc;
    {   // inside a stream capture (CUDA graph) nothing may be allocated and nothing is read back: the buffers must be
        // there already (gx_reserve, or one ordinary call of the same shape), and the graph replays the rounds of
        // stage kernels the handle's history asks for at capture time (the tail kernel still renders any wave beyond)
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        GX_CUDA(cudaStreamIsCapturing(stream, &cs));
        sc->capturing = cs == cudaStreamCaptureStatusActive;
        if (sc->capturing && sc->opt_timing) return fail(GX_ERR_UNSUPPORTED, "option \"timing\" cannot be used during stream capture");
    }
    if ((rc = setup_buffers(sc, PP, worst_tris)) != GX_OK) return rc;
    sc->last_stream = stream;
    if (st) GX_CUDA(cudaMemsetAsync(sc->stats, 0, GX_NSTAT * sizeof(unsigned long long), stream));
    GX_CUDA(cudaMemsetAsync(PP.ctl, 0, 64 * sizeof(uint32_t), stream));
    if (PP.occl) GX_CUDA(cudaMemsetAsync(PP.hizt, 0, (size_t)N * (size_t)PP.hz_stride * sizeof(uint32_t), stream));
    if ((rc = mark(sc, stream, 0)) != GX_OK) return rc;

    // K1: one CTA per environment: 4 warps for small scenes, 16 where an environment has thousands of sub-clusters
    {
        const size_t csmem = gx::env_smem_bytes(K);
        if ((size_t)PP.item_stride > 512) {
            auto ck = st ? gx::cull_kernel<16, true> : gx::cull_kernel<16, false>;
            ck<<<N, 16 * 32, csmem, stream>>>(PP);
        } else {
            auto ck = st ? gx::cull_kernel<4, true> : gx::cull_kernel<4, false>;
            ck<<<N, 4 * 32, csmem, stream>>>(PP);
        }
        GX_CUDA(cudaGetLastError());
        if ((rc = mark(sc, stream, 1)) != GX_OK) return rc;
    }
    int launches = 1;
    // one round of the stage kernels per wave the previous call on this handle needed (its batch is the best guess
    // for this one), plus one when there were several; whatever is still left goes to the cooperative tail kernel
    int rounds = sc->hist_waves > 1 ? sc->hist_waves + 1 : 1;
    if (sc->opt_max_rounds > 0) rounds = std::min(rounds, sc->opt_max_rounds);
    for (int round = 0; round < rounds; ++round) {
    if (round > 0) {
        gx::wave_kernel<<<1, 256, 0, stream>>>(PP);
        GX_CUDA(cudaGetLastError());
        ++launches;
    }
    gx::pack_kernel<<<std::min(std::max(N / 8, 1), 4 * sc->num_sms), 256, 0, stream>>>(PP);
    GX_CUDA(cudaGetLastError());
    if ((rc = mark(sc, stream, round > 0 ? 5 : 1)) != GX_OK) return rc;
    ++launches;
    for (int phase = PP.occl ? 1 : 0; phase <= (PP.occl ? 2 : 0); ++phase) {
        if (phase == 2) {   // the runs of the second phase against the hi-Z pyramid of the first, densely
            auto ck = st ? gx::cull2_kernel<true> : gx::cull2_kernel<false>;
            ck<<<sc->num_sms * 4, 256, 0, stream>>>(PP);
            GX_CUDA(cudaGetLastError());
            if ((rc = mark(sc, stream, 1)) != GX_OK) return rc;
            ++launches;
        }
        // K2: persistent independent warps
        {
            constexpr int GW = 8;
            const bool hz = phase == 2 && PP.hiz;
            auto gk = hz ? (st ? gx::geom_kernel<GW, true, true> : gx::geom_kernel<GW, false, true>)
                         : (st ? gx::geom_kernel<GW, true, false> : gx::geom_kernel<GW, false, false>);
            const size_t gsmem = (size_t)GW * gx::GEOM_WARP_SMEM;
            int per_sm = 0;
            if ((rc = plan_of(sc, (const void *)gk, GW * 32, gsmem, &per_sm)) != GX_OK) return rc;
            if (sc->opt_ctas_per_sm) per_sm = std::min(per_sm, sc->opt_ctas_per_sm);
            gk<<<sc->num_sms * per_sm, GW * 32, gsmem, stream>>>(PP, phase);
            GX_CUDA(cudaGetLastError());
            if ((rc = mark(sc, stream, 2)) != GX_OK) return rc;
        }
        // K3: one CTA per environment at a time
        {
            auto bk = st ? gx::bin_kernel<true> : gx::bin_kernel<false>;
            const size_t bsmem = (size_t)2 * PP.T * gx::NBUCKET * 4;
            int per_sm = 0;
            // (thread t of the CTA owns tile t in the scan, so a CTA has at least T = 256 threads at the largest frame)
            const int bthreads = sc->opt_bin_threads ? sc->opt_bin_threads : 512;
            if ((rc = plan_of(sc, (const void *)bk, bthreads, bsmem, &per_sm)) != GX_OK) return rc;
            bk<<<std::min(N, sc->num_sms * per_sm), bthreads, bsmem, stream>>>(PP, phase);
            GX_CUDA(cudaGetLastError());
            if ((rc = mark(sc, stream, 3)) != GX_OK) return rc;
        }
        // K4 + K5: persistent independent warps, one tile each at a time
        {
            constexpr int RW = 8;
            auto rk = phase == 0 ? (st ? gx::raster_kernel<RW, true, 0> : gx::raster_kernel<RW, false, 0>)
                    : phase == 1 ? (st ? gx::raster_kernel<RW, true, 1> : gx::raster_kernel<RW, false, 1>)
                                 : (st ? gx::raster_kernel<RW, true, 2> : gx::raster_kernel<RW, false, 2>);
            const size_t rsmem = (size_t)RW * gx::RAST_WARP_SMEM;
            int per_sm = 0;
            if ((rc = plan_of(sc, (const void *)rk, RW * 32, rsmem, &per_sm)) != GX_OK) return rc;
            if (sc->opt_ctas_per_sm) per_sm = std::min(per_sm, sc->opt_ctas_per_sm);
            rk<<<sc->num_sms * per_sm, RW * 32, rsmem, stream>>>(PP);
            GX_CUDA(cudaGetLastError());
            if ((rc = mark(sc, stream, 4)) != GX_OK) return rc;
        }
        launches += 3;
    }
    }
    // the tail: later waves, on the device (exits at once when the first wave took every environment)
    {
        auto tk = st ? gx::tail_kernel<true> : gx::tail_kernel<false>;
        const size_t tsmem = gx::tail_smem_bytes(PP.T);
        int per_sm = 0;
        if ((rc = plan_of(sc, (const void *)tk, gx::TAIL_WARPS * 32, tsmem, &per_sm)) != GX_OK) return rc;
        void *args[1] = {(void *)&PP};
        GX_CUDA(cudaLaunchCooperativeKernel((const void *)tk, dim3((unsigned)(sc->num_sms * per_sm)), dim3(gx::TAIL_WARPS * 32), args, tsmem, stream));
        if ((rc = mark(sc, stream, 5)) != GX_OK) return rc;
    }
    if (!sc->ctl_pending && !sc->capturing) {   // (a read-back still in flight keeps its buffer)
        GX_CUDA(cudaMemcpyAsync(sc->h_ctl, PP.ctl, gx::C_NCTL * sizeof(uint32_t), cudaMemcpyDeviceToHost, stream));
        GX_CUDA(cudaEventRecord(sc->ev_ctl, stream));
        sc->ctl_pending = true;
        sc->ctl_N = N;
    }
    sc->last_launches = launches + 1;
    if (sc->opt_timing && !sc->t_full) ++sc->t_calls;
    return GX_OK;
}

int gx_reserve(GxScene *sc, const GxCamera *cam, int32_t N, int32_t K) {
    if (!sc || !cam) return fail(GX_ERR_INVALID_ARG, "NULL scene or camera");
    if (N <= 0 || K < 0 || K > GX_MAX_INSTANCES) return fail(GX_ERR_INVALID_ARG, "bad N or K");
    if (cam->width <= 0 || cam->height <= 0 || cam->width % 16 || cam->height % 16 || cam->width > GX_MAX_FRAME || cam->height > GX_MAX_FRAME)
        return fail(GX_ERR_INVALID_ARG, "width and height must be positive multiples of 16 up to %d", GX_MAX_FRAME);
    DeviceGuard guard(sc->device);
    if (!guard.ok) return fail(GX_ERR_CUDA, "cannot select CUDA device %d", sc->device);
    sc->capturing = false;
    gx::PipeParams PP;
    memset(&PP, 0, sizeof(PP));
    PP.g.N = N; PP.g.K = K; PP.g.W = cam->width; PP.g.H = cam->height;
    PP.tiles_x = cam->width / gx::TILE; PP.tiles_y = cam->height / gx::TILE; PP.T = PP.tiles_x * PP.tiles_y;
    PP.occl = sc->opt_hiz && (sc->opt_occlusion == 1 || (sc->opt_occlusion < 0 && cam->width * cam->height >= 4096)) ? 1 : 0;
    const unsigned long long worst_tris = (unsigned long long)sc->max_static_nt + (unsigned long long)K * sc->max_dyn_nt;
    return setup_buffers(sc, PP, worst_tris);
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

int gx_set_robot(GxScene *sc, const GxLink *links, int32_t n_links, int32_t camera_link, const float *cam_mount, int32_t ee_link) {
    if (!sc || !links || !cam_mount) return fail(GX_ERR_INVALID_ARG, "NULL argument");
    if (n_links <= 0 || n_links > gx::FK_MAX_LINKS) return fail(GX_ERR_INVALID_ARG, "n_links must be in [1, %d], got %d", gx::FK_MAX_LINKS, n_links);
    if (camera_link < -1 || camera_link >= n_links || ee_link < -1 || ee_link >= n_links)
        return fail(GX_ERR_INVALID_ARG, "camera_link and ee_link must be in [-1, n_links)");
    std::vector<gx::FkLink> h((size_t)n_links);
    for (int l = 0; l < n_links; ++l) {
        if (links[l].parent < -1 || links[l].parent >= l) return fail(GX_ERR_INVALID_ARG, "link %d: parent %d must precede it (or be -1)", l, links[l].parent);
        if (links[l].joint_type < 0 || links[l].joint_type > 2) return fail(GX_ERR_INVALID_ARG, "link %d: joint_type %d", l, links[l].joint_type);
        h[l].parent = links[l].parent;
        h[l].joint_type = links[l].joint_type;
        memcpy(h[l].axis, links[l].axis, sizeof(h[l].axis));
        memcpy(h[l].origin, links[l].origin, sizeof(h[l].origin));
    }
    DeviceGuard guard(sc->device);
    if (!guard.ok) return fail(GX_ERR_CUDA, "cannot select CUDA device %d", sc->device);
    if (sc->fk_links) { cudaFree(sc->fk_links); sc->fk_links = nullptr; sc->fk_L = 0; }
    GX_CUDA(cudaMalloc(&sc->fk_links, (size_t)n_links * sizeof(gx::FkLink)));
    GX_CUDA(cudaMemcpy(sc->fk_links, h.data(), (size_t)n_links * sizeof(gx::FkLink), cudaMemcpyHostToDevice));
    sc->fk_L = n_links;
    sc->fk_camera_link = camera_link;
    sc->fk_ee_link = ee_link;
    memcpy(sc->fk_mount, cam_mount, sizeof(sc->fk_mount));
    return GX_OK;
}

int gx_update_transforms(GxScene *sc, int32_t N, int32_t K, int32_t link_slot0, const float *base_pose, const float *joint_pos,
                         const int32_t *held_slot, const float *held_xform, float *cam_pose, float *inst_xform, void *cuda_stream) {
    if (!sc) return fail(GX_ERR_INVALID_ARG, "NULL scene");
    if (!sc->fk_links) return fail(GX_ERR_INVALID_ARG, "no robot: call gx_set_robot first");
    if (N <= 0 || K < 0 || K > GX_MAX_INSTANCES) return fail(GX_ERR_INVALID_ARG, "bad N or K");
    if (!base_pose || !joint_pos || !cam_pose || !inst_xform) return fail(GX_ERR_INVALID_ARG, "NULL array argument");
    if ((held_slot == nullptr) != (held_xform == nullptr)) return fail(GX_ERR_INVALID_ARG, "held_slot and held_xform go together");
    if (link_slot0 < 0 || link_slot0 + sc->fk_L > K) return fail(GX_ERR_INVALID_ARG, "link slots [%d, %d) do not fit K = %d", link_slot0, link_slot0 + sc->fk_L, K);
    DeviceGuard guard(sc->device);
    if (!guard.ok) return fail(GX_ERR_CUDA, "cannot select CUDA device %d", sc->device);
    gx::FkParams P;
    P.links = sc->fk_links; P.L = sc->fk_L; P.camera_link = sc->fk_camera_link; P.ee_link = sc->fk_ee_link;
    memcpy(P.cam_mount, sc->fk_mount, sizeof(P.cam_mount));
    P.N = N; P.K = K; P.link_slot0 = link_slot0;
    P.base_pose = base_pose; P.joint_pos = joint_pos; P.held_slot = held_slot; P.held_xform = held_xform;
    P.cam_pose = cam_pose; P.inst_xform = inst_xform;
    constexpr int FW = 4;
    gx::fk_kernel<FW><<<(N + FW - 1) / FW, FW * 32, 0, (cudaStream_t)cuda_stream>>>(P);
    GX_CUDA(cudaGetLastError());
    return GX_OK;
}

int gx_set_collision_world(GxScene *sc, const GxColumnGrid *grids, int32_t n_radii, const float *radii, const GxSphere *spheres,
                           int32_t n_spheres) {
    if (!sc || !grids || !radii || !spheres) return fail(GX_ERR_INVALID_ARG, "NULL argument");
    if (n_radii <= 0 || n_radii > 16 || n_spheres <= 0 || n_spheres > 4096) return fail(GX_ERR_INVALID_ARG, "bad n_radii or n_spheres");
    const size_t ng = (size_t)sc->n_static * (size_t)n_radii;
    std::vector<gx::ColGridDev> hg(ng);
    std::vector<uint32_t> hoff;
    std::vector<float2> hlay;
    for (size_t i = 0; i < ng; ++i) {
        const GxColumnGrid &g = grids[i];
        if (g.nx <= 0 || g.nz <= 0 || !(g.spacing > 0.0f) || !g.col_off || (unsigned long long)g.nx * g.nz >= (1ull << 30))
            return fail(GX_ERR_INVALID_ARG, "column grid %zu: bad size, spacing or NULL col_off", i);
        const size_t nc = (size_t)g.nx * g.nz;
        const uint32_t nl = g.col_off[nc];
        if (nl && !g.layers) return fail(GX_ERR_INVALID_ARG, "column grid %zu: NULL layers", i);
        for (size_t c = 0; c < nc; ++c)
            if (g.col_off[c] > g.col_off[c + 1]) return fail(GX_ERR_INVALID_ARG, "column grid %zu: col_off not ascending", i);
        if (hoff.size() + nc + 1 >= 0xFFFFFFFFull || hlay.size() + nl >= 0xFFFFFFFFull) return fail(GX_ERR_UNSUPPORTED, "column grids too large");
        hg[i] = {g.x0, g.z0, g.spacing, g.nx, g.nz, (uint32_t)hoff.size(), (uint32_t)hlay.size(), 0u};
        hoff.insert(hoff.end(), g.col_off, g.col_off + nc + 1);
        for (uint32_t l = 0; l < nl; ++l) hlay.push_back(make_float2(g.layers[2 * (size_t)l], g.layers[2 * (size_t)l + 1]));
    }
    std::vector<gx::SphereDev> hs((size_t)n_spheres);
    int max_link = -1;
    for (int i = 0; i < n_spheres; ++i) {
        if (spheres[i].link < -1 || spheres[i].radius_class < 0 || spheres[i].radius_class >= n_radii)   // (-1: on the grasped object)
            return fail(GX_ERR_INVALID_ARG, "sphere %d: bad link or radius class", i);
        hs[i] = {spheres[i].link, spheres[i].radius_class, spheres[i].centre[0], spheres[i].centre[1], spheres[i].centre[2]};
        max_link = std::max(max_link, spheres[i].link);
    }
    DeviceGuard guard(sc->device);
    if (!guard.ok) return fail(GX_ERR_CUDA, "cannot select CUDA device %d", sc->device);
    cudaFree(sc->cg_grids); cudaFree(sc->cg_col_off); cudaFree(sc->cg_layers); cudaFree(sc->cg_radii); cudaFree(sc->cg_spheres);
    sc->cg_grids = nullptr; sc->cg_col_off = nullptr; sc->cg_layers = nullptr; sc->cg_radii = nullptr; sc->cg_spheres = nullptr;
    sc->cg_S = 0;
    int rc;
    std::vector<float> hr(radii, radii + n_radii);
    if ((rc = upload(sc->cg_grids, hg)) != GX_OK || (rc = upload(sc->cg_col_off, hoff)) != GX_OK || (rc = upload(sc->cg_layers, hlay)) != GX_OK ||
        (rc = upload(sc->cg_radii, hr)) != GX_OK || (rc = upload(sc->cg_spheres, hs)) != GX_OK)
        return rc;
    sc->cg_n_radii = n_radii;
    sc->cg_S = n_spheres;
    sc->cg_max_link = max_link;
    return GX_OK;
}

int gx_collide_batch(GxScene *sc, int32_t N, int32_t K, const int32_t *env_scene, const int32_t *inst_mesh, const float *inst_xform,
                     int32_t link_slot0, int32_t obj_slot0, int32_t n_obj, const int32_t *held_slot, uint8_t *out_static,
                     int32_t *out_object, void *cuda_stream) {
    if (!sc) return fail(GX_ERR_INVALID_ARG, "NULL scene");
    if (!sc->cg_S) return fail(GX_ERR_INVALID_ARG, "no collision world: call gx_set_collision_world first");
    if (N <= 0 || K <= 0 || K > GX_MAX_INSTANCES) return fail(GX_ERR_INVALID_ARG, "bad N or K");
    if (!env_scene || !inst_xform || !out_static || !out_object || (n_obj > 0 && !inst_mesh)) return fail(GX_ERR_INVALID_ARG, "NULL array argument");
    if (link_slot0 < 0 || link_slot0 + sc->cg_max_link >= K) return fail(GX_ERR_INVALID_ARG, "link slots do not fit K = %d", K);
    if (obj_slot0 < 0 || n_obj < 0 || obj_slot0 + n_obj > K) return fail(GX_ERR_INVALID_ARG, "object slots [%d, %d) do not fit K = %d", obj_slot0, obj_slot0 + n_obj, K);
    DeviceGuard guard(sc->device);
    if (!guard.ok) return fail(GX_ERR_CUDA, "cannot select CUDA device %d", sc->device);
    gx::CollideParams P;
    P.grids = sc->cg_grids; P.col_off = sc->cg_col_off; P.layers = sc->cg_layers; P.radii = sc->cg_radii; P.spheres = sc->cg_spheres;
    P.mesh_box = sc->mesh_box;
    P.n_static = sc->n_static; P.n_radii = sc->cg_n_radii; P.n_dyn = sc->n_dyn; P.S = sc->cg_S;
    P.N = N; P.K = K; P.link_slot0 = link_slot0; P.obj_slot0 = obj_slot0; P.n_obj = n_obj;
    P.env_scene = env_scene; P.inst_mesh = inst_mesh; P.inst_xform = inst_xform; P.held_slot = held_slot;
    P.out_static = out_static; P.out_object = out_object;
    constexpr int CW = 4;
    gx::collide_kernel<CW><<<(N + CW - 1) / CW, CW * 32, 0, (cudaStream_t)cuda_stream>>>(P);
    GX_CUDA(cudaGetLastError());
    return GX_OK;
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
    if (!sc->copy_stream) GX_CUDA(cudaStreamCreateWithFlags(&sc->copy_stream, cudaStreamNonBlocking));
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
    // render in sub-batches and copy each one's images back on a second stream while the next one renders.  The
    // device-to-host copy of RGBD over PCIe takes about twice as long as the rendering, and a render call has a
    // fixed cost of a few hundred microseconds, so three sub-batches are the best split measured on cfg 2
    // (time = first render + the whole copy): 2.76 ms against 2.09 ms for the bare copy at 56 GB/s.
    const int sub = sc->opt_host_sub > 0 ? sc->opt_host_sub : std::max(64, (N + 2) / 3);
    size_t n_sub = 0;
    for (int e0 = 0; e0 < N; e0 += sub, ++n_sub) {
        const int n = std::min(sub, N - e0);
        const size_t o = (size_t)e0 * npix, cnt = (size_t)n * npix;
        rc = gx_render_batch(sc, cam, n, K, sc->h_env_scene.p + e0, sc->h_cam_pose.p + (size_t)e0 * 16,
                             K > 0 ? sc->h_inst_mesh.p + (size_t)e0 * K : nullptr,
                             K > 0 ? sc->h_inst_xform.p + (size_t)e0 * K * 16 : nullptr,
                             rgb_out ? sc->h_rgb.p + o * 3 : nullptr, sc->h_depth.p + o, id_out ? sc->h_id.p + o : nullptr, st);
        if (rc != GX_OK) return rc;
        if (n_sub == sc->ev_sub.size()) {
            cudaEvent_t e;
            GX_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            sc->ev_sub.push_back(e);
        }
        GX_CUDA(cudaEventRecord(sc->ev_sub[n_sub], st));
        GX_CUDA(cudaStreamWaitEvent(sc->copy_stream, sc->ev_sub[n_sub], 0));
        GX_CUDA(cudaMemcpyAsync(depth_out + o, sc->h_depth.p + o, cnt * 4, cudaMemcpyDeviceToHost, sc->copy_stream));
        if (rgb_out) GX_CUDA(cudaMemcpyAsync(rgb_out + o * 3, sc->h_rgb.p + o * 3, cnt * 3, cudaMemcpyDeviceToHost, sc->copy_stream));
        if (id_out) GX_CUDA(cudaMemcpyAsync(id_out + o, sc->h_id.p + o, cnt * 4, cudaMemcpyDeviceToHost, sc->copy_stream));
    }
    GX_CUDA(cudaStreamSynchronize(sc->copy_stream));
    GX_CUDA(cudaStreamSynchronize(st));
    return GX_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// gx_render_batch_noalloc (include/gx.h): the render path for callers that must not enter the CUDA allocator.
// Everything gx_render_batch keeps in cudaMalloc'ed buffers of the handle (record arena, per-call tables) lives in
// the array below instead, which belongs to the library's device image: it exists on every GPU that loads these
// kernels, from module load to process exit, and no call ever allocates or frees it.
// ------------------------------------------------------------------------------------------------
namespace {

// The scratch.  In HOST code this name is only a handle for the runtime's symbol calls -- it is not a device address,
// and a kernel handed `g_noalloc_scratch` from the host would fault (or, on a system where the GPU can reach host
// memory, quietly use host memory).  The host gets the real address once per device from cudaGetSymbolAddress
// (noalloc_device_setup) and passes that to the kernels inside PipeParams.
static __device__ __align__(256) unsigned char g_noalloc_scratch[GX_NOALLOC_SCRATCH_BYTES];

// K2-K5 over the whole batch as ONE cooperative kernel: tail_kernel's wave loop (gx_pipeline.cuh), except that it
// starts at environment 0 instead of where the host-launched first wave ended.  cull_kernel has run before it on the
// same stream (U, item lists and model-view tables are in the scratch); its own allocation of a first wave is simply
// redone here.
__global__ void __launch_bounds__(gx::TAIL_WARPS * 32, 3) noalloc_waves_kernel(const gx::PipeParams PP) {
    using namespace gx;
    extern __shared__ __align__(16) unsigned char smem[];
    cg::grid_group grid = cg::this_grid();
    const int warp = threadIdx.x >> 5;
    uint32_t e_next = 0;
    while (e_next < (uint32_t)PP.g.N) {
        grid.sync();   // every CTA has read the end of the previous wave before the control words change
        if (blockIdx.x == 0) alloc_wave(PP, e_next);
        grid.sync();
        pack_stage<true>(PP);
        grid.sync();
        for (int phase = PP.occl ? 1 : 0; phase <= (PP.occl ? 2 : 0); ++phase) {
            if (phase == 2) {
                cull2_stage<true, false>(PP);
                grid.sync();
            }
            if (phase == 2 && PP.hiz) geom_stage<true, false, true>(PP, smem + (size_t)warp * GEOM_WARP_SMEM, phase);
            else geom_stage<true, false, false>(PP, smem + (size_t)warp * GEOM_WARP_SMEM, phase);
            grid.sync();
            bin_stage<true, false>(PP, reinterpret_cast<uint32_t *>(smem), reinterpret_cast<uint32_t *>(smem) + PP.T * NBUCKET, phase);
            grid.sync();
            if (phase == 0) raster_stage<true, false, 0>(PP, smem + (size_t)warp * RAST_WARP_SMEM);
            else if (phase == 1) raster_stage<true, false, 1>(PP, smem + (size_t)warp * RAST_WARP_SMEM);
            else raster_stage<true, false, 2>(PP, smem + (size_t)warp * RAST_WARP_SMEM);
            grid.sync();
        }
        e_next = __ldcg(&PP.ctl[C_WAVE_E1]);
    }
}

// What the first call on a device finds out and every later call reuses.  Plain static storage: nothing is allocated.
constexpr int NOALLOC_MAX_DEVICES = 64;
struct NoallocDevice {
    bool ready = false;
    unsigned char *base = nullptr;   // device address of g_noalloc_scratch on this device
    int ctas_per_sm = 0;             // co-resident CTAs of noalloc_waves_kernel at its largest shared-memory size
};
NoallocDevice g_noalloc_dev[NOALLOC_MAX_DEVICES];
std::mutex g_noalloc_mutex;

// Once per device, with that device current (the caller's DeviceGuard): the array's address on THIS device -- each
// device has its own copy of the array at its own address -- and the cooperative kernel's launch shape.
int noalloc_device_setup(int device, NoallocDevice **out) {
    if (device < 0 || device >= NOALLOC_MAX_DEVICES)
        return fail(GX_ERR_UNSUPPORTED, "gx_render_batch_noalloc supports device ordinals below %d, got %d", NOALLOC_MAX_DEVICES, device);
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    NoallocDevice &d = g_noalloc_dev[device];
    if (!d.ready) {
        int coop = 0;
        GX_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, device));
        if (!coop) return fail(GX_ERR_UNSUPPORTED, "device %d cannot launch cooperative kernels", device);
        void *p = nullptr;
        GX_CUDA(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p || ((uintptr_t)p & 255u)) return fail(GX_ERR_CUDA, "cudaGetSymbolAddress gave %p for the scratch array", p);
        const size_t smem = gx::tail_smem_bytes((GX_MAX_FRAME / gx::TILE) * (GX_MAX_FRAME / gx::TILE));   // (the largest any frame needs)
        GX_CUDA(cudaFuncSetAttribute((const void *)noalloc_waves_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int per_sm = 0;
        GX_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)noalloc_waves_kernel, gx::TAIL_WARPS * 32, smem));
        if (per_sm < 1) return fail(GX_ERR_UNSUPPORTED, "the cooperative kernel does not fit an SM of device %d", device);
        d.base = static_cast<unsigned char *>(p);
        d.ctas_per_sm = per_sm;
        d.ready = true;
    }
    *out = &d;
    return GX_OK;
}

}  // namespace

extern "C" int gx_render_batch_noalloc(GxScene *sc, const GxCamera *cam, int32_t N, int32_t K, const int32_t *env_scene,
                                       const float *cam_pose, const int32_t *inst_mesh, const float *inst_xform,
                                       uint8_t *rgb_out, float *depth_out, uint32_t *id_out, void *cuda_stream) {
    if (!sc || !cam) return fail(GX_ERR_INVALID_ARG, "NULL scene or camera");
    if (N <= 0) return fail(GX_ERR_INVALID_ARG, "N must be positive, got %d", N);
    if (K < 0 || K > GX_MAX_INSTANCES) return fail(GX_ERR_INVALID_ARG, "K must be in [0, %d], got %d", GX_MAX_INSTANCES, K);
    if (!env_scene || !cam_pose || !depth_out) return fail(GX_ERR_INVALID_ARG, "env_scene, cam_pose and depth_out are required");
    if (K > 0 && (!inst_mesh || !inst_xform)) return fail(GX_ERR_INVALID_ARG, "inst_mesh and inst_xform are required when K > 0");
    if (cam->width <= 0 || cam->height <= 0 || cam->width % 16 || cam->height % 16)
        return fail(GX_ERR_INVALID_ARG, "width and height must be positive multiples of 16, got %dx%d", cam->width, cam->height);
    if (!(cam->znear > 0.0f) || !(cam->zfar > cam->znear)) return fail(GX_ERR_INVALID_ARG, "need 0 < znear < zfar");
    if (!(cam->fx > 0.0f) || !(cam->fy > 0.0f)) return fail(GX_ERR_INVALID_ARG, "fx and fy must be positive");
    if (cam->width > GX_MAX_FRAME || cam->height > GX_MAX_FRAME)
        return fail(GX_ERR_UNSUPPORTED, "width and height must be <= %d, got %dx%d", GX_MAX_FRAME, cam->width, cam->height);
    const unsigned long long worst_tris = (unsigned long long)sc->max_static_nt + (unsigned long long)K * sc->max_dyn_nt;
    if (worst_tris >= (1ull << 29)) return fail(GX_ERR_UNSUPPORTED, "more than 2^29 triangles per environment");
    DeviceGuard guard(sc->device);
    if (!guard.ok) return fail(GX_ERR_CUDA, "cannot select CUDA device %d", sc->device);
    NoallocDevice *dev = nullptr;
    int rc;
    if ((rc = noalloc_device_setup(sc->device, &dev)) != GX_OK) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;

    gx::PipeParams PP;
    memset(&PP, 0, sizeof(PP));
    GxParams &P = PP.g;
    P.verts = sc->verts; P.tris = sc->tris; P.batches = sc->batches; P.subs = sc->subs; P.clusters = sc->clusters; P.meshes = sc->meshes;
    P.n_static = sc->n_static; P.n_dyn = sc->n_dyn;
    P.N = N; P.K = K; P.W = cam->width; P.H = cam->height;
    P.fx = cam->fx; P.fy = cam->fy; P.znear = cam->znear; P.zfar = cam->zfar;
    P.env_scene = env_scene; P.cam_pose = cam_pose; P.inst_mesh = inst_mesh; P.inst_xform = inst_xform;
    P.rgb = rgb_out; P.depth = depth_out; P.id = id_out;
    P.obs = nullptr; P.obs_dmin = 0.0f; P.obs_dmax = 1.0f; P.obs_range = 1.0f;
    P.stats = sc->stats;   // (never touched: only the kernels without the statistics are used here)
    P.cull = sc->opt_cull;
    PP.tiles_x = P.W / gx::TILE; PP.tiles_y = P.H / gx::TILE; PP.T = PP.tiles_x * PP.tiles_y;
    PP.bucket_off = -log2f(P.znear);
    PP.bucket_scale = (float)gx::NBUCKET / log2f(P.zfar / P.znear);
    PP.subcull = sc->opt_subcull;
    PP.big_px = sc->opt_big_px;
    PP.hiz = sc->opt_hiz;
    PP.occl = sc->opt_hiz && (sc->opt_occlusion == 1 || (sc->opt_occlusion < 0 && P.W * P.H >= 4096)) ? 1 : 0;
    PP.occl_area = (float)sc->opt_occl_area;
    PP.item_stride = (int32_t)std::max<size_t>((size_t)sc->max_static_batches + (size_t)K * sc->max_dyn_batches, 1);
    PP.hz_stride = 0;
    for (int w = PP.tiles_x, h = PP.tiles_y;; w = (w + 1) >> 1, h = (h + 1) >> 1) { PP.hz_stride += w * h; if (w == 1 && h == 1) break; }

    // ---- carve the array: tables first (the order of setup_buffers), the arena takes what is left ------------
    const size_t cap = (size_t)GX_NOALLOC_SCRATCH_BYTES;
    const size_t n = (size_t)N, k1 = (size_t)K + 1, NK1 = (size_t)PP.T * gx::NBUCKET + 1, istr = (size_t)PP.item_stride;
    size_t off = 0;   // bytes
    auto take = [&off](size_t bytes) { const size_t at = off; off = (off + bytes + 255) & ~(size_t)255; return at; };   // (N < 2^31 and the factors below keep every product far inside 64 bits)
    const size_t o_ctl = take(64 * 4);
    const size_t o_U = take(n * 4), o_nitems = take(n * 4), o_cpre = take((n + 1) * 4), o_base = take(n * 4);
    const size_t o_cnt = take(n * 4), o_cntA = take(n * 4), o_nl = take(n * 4);
    const size_t o_idb = take(n * k1 * 4), o_mv = take(n * k1 * 48);
    const size_t o_toff = take(n * NK1 * 4), o_tasks = take((size_t)gx::NCLASS * n * (size_t)PP.T * 4);
    const size_t hizt_bytes = PP.occl ? n * (size_t)PP.hz_stride * 4 : 0;
    const size_t o_hizt = take(hizt_bytes), o_hizb = take(PP.occl ? n * (size_t)PP.T * 32 : 0);
    const size_t o_items = take(n * istr * 16), o_witems = take(n * istr * 16), o_witems2 = take(PP.occl ? n * istr * 16 : 0);
    const size_t o_keys = take(PP.occl ? n * (size_t)P.W * (size_t)P.H * 8 : 0);
    const size_t tables = off;
    // record slots: 64 bytes of record, 8 of box / depth word, 16 of tile references; the arena must hold the largest
    // environment the scene can produce (setup_buffers has the reasoning), more only shortens the wave loop
    const unsigned long long worst_env = 4ull * worst_tris + 64;
    const unsigned long long need = (unsigned long long)tables + worst_env * 88ull + 3 * 256;
    if (need > cap)
        return fail(GX_ERR_UNSUPPORTED, "gx_render_batch_noalloc: N = %d, K = %d at %dx%d needs %llu bytes of scratch (%zu for the tables of "
                    "the call, the rest for an arena of one worst-case environment of %llu triangles) but the built-in array holds "
                    "GX_NOALLOC_SCRATCH_BYTES = %zu; render fewer environments per call, or use gx_render_batch where allocation is allowed",
                    N, K, cam->width, cam->height, need, tables, worst_tris, cap);
    unsigned long long slots = (cap - tables - 3 * 256) / 88ull;
    slots = std::min<unsigned long long>(slots, std::min<unsigned long long>((unsigned long long)N * worst_env, 0xFFFFFF00ull));
    const size_t o_recs = take((size_t)slots * 64), o_bbs = take((size_t)slots * 8), o_refs = take((size_t)slots * 16);
    if (off > cap) return fail(GX_ERR_UNSUPPORTED, "gx_render_batch_noalloc: internal layout error (%zu > %zu bytes)", off, cap);
    unsigned char *b = dev->base;
    PP.ctl = reinterpret_cast<uint32_t *>(b + o_ctl); PP.U = reinterpret_cast<uint32_t *>(b + o_U);
    PP.n_items = reinterpret_cast<uint32_t *>(b + o_nitems); PP.item_pre = reinterpret_cast<uint32_t *>(b + o_cpre);
    PP.rec_base = reinterpret_cast<uint32_t *>(b + o_base); PP.cnt = reinterpret_cast<uint32_t *>(b + o_cnt);
    PP.cntA = reinterpret_cast<uint32_t *>(b + o_cntA); PP.n_large = reinterpret_cast<uint32_t *>(b + o_nl);
    PP.env_idb = reinterpret_cast<uint32_t *>(b + o_idb); PP.env_mv = reinterpret_cast<float *>(b + o_mv);
    PP.tile_off = reinterpret_cast<uint32_t *>(b + o_toff); PP.tasks = reinterpret_cast<uint32_t *>(b + o_tasks);
    PP.hizt = reinterpret_cast<uint32_t *>(b + o_hizt); PP.hizb = reinterpret_cast<uint32_t *>(b + o_hizb);
    PP.items = reinterpret_cast<uint4 *>(b + o_items); PP.wave_items = reinterpret_cast<uint4 *>(b + o_witems);
    PP.wave_items2 = reinterpret_cast<uint4 *>(b + o_witems2);
    PP.keys = reinterpret_cast<unsigned long long *>(b + o_keys);
    PP.recs = reinterpret_cast<uint4 *>(b + o_recs); PP.bbs = reinterpret_cast<uint2 *>(b + o_bbs);
    PP.refs = reinterpret_cast<uint32_t *>(b + o_refs);
    PP.arena_slots = (uint32_t)slots;

    // ---- what must start at zero; everything else in the array is written before it is read -------------------
    GX_CUDA(cudaMemsetAsync(PP.ctl, 0, 64 * sizeof(uint32_t), stream));
    if (PP.occl) GX_CUDA(cudaMemsetAsync(PP.hizt, 0, hizt_bytes, stream));
    // K1, as in gx_render_batch
    {
        const size_t csmem = gx::env_smem_bytes(K);
        if ((size_t)PP.item_stride > 512) gx::cull_kernel<16, false><<<N, 16 * 32, csmem, stream>>>(PP);
        else gx::cull_kernel<4, false><<<N, 4 * 32, csmem, stream>>>(PP);
        GX_CUDA(cudaGetLastError());
    }
    // K2-K5, all waves
    {
        int per_sm = dev->ctas_per_sm;
        if (sc->opt_ctas_per_sm) per_sm = std::min(per_sm, sc->opt_ctas_per_sm);
        void *args[1] = {(void *)&PP};
        GX_CUDA(cudaLaunchCooperativeKernel((const void *)noalloc_waves_kernel, dim3((unsigned)(sc->num_sms * per_sm)),
                                            dim3(gx::TAIL_WARPS * 32), args, gx::tail_smem_bytes(PP.T), stream));
    }
    return GX_OK;
}
