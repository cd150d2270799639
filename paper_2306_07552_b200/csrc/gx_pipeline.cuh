// gx_pipeline.cuh -- the render path of gx_render_batch (sm_100a), DESIGN.md section 5:
//
//   cull_kernel    K1   per environment: cluster AABBs against the frustum, then the 32-triangle sub-clusters of
//                       the survivors; one 16-byte work item per batch that has a run of triangles left, in the
//                       environment's own item segment, and U[env] = an upper bound of the record slots the
//                       environment can produce.  The last CTA to finish runs alloc_wave: an exclusive scan of U
//                       over the environments gives every environment of the wave its exact segment of the
//                       record arena, so no segment can overflow.
//   geom_kernel    K2   vertex transform / near clip / snap / set-up (N1-N6).  Independent warps, no CTA-level
//                       synchronisation; one 64-byte record per surviving triangle (two slots for a near-clipped
//                       piece: record + float colours).  Records whose pixel box fits a 16x16 square ("small") grow
//                       from the bottom of the segment, the others ("large") from its top.
//   bin_kernel     K3   per environment: count -> exclusive scan -> fill of the small records into per-(tile,
//                       depth bucket) lists of record indices (16x16-pixel tiles; the bucket of the nearest vertex
//                       orders a tile's list front to back); exact sizes, nothing can overflow.  Also files every
//                       tile as a raster task under its cost class.
//   raster_kernel  K4+K5  persistent independent warps; a task is one tile of one environment and the warp OWNS
//                       the tile's 256 (depth, record) keys in shared memory: large records first, pixel-parallel in
//                       8x4-pixel blocks with a block-level trivial reject and a live hi-Z value per block (plain
//                       compare-and-store, no atomics); then the tile's small records, front to back, skipped when
//                       hidden behind the hi-Z values, their boxes cut into 4-pixel slots dealt evenly to the lanes;
//                       finally the winner's colour is resolved from its record and RGB / depth / id (or the packed
//                       observation) leave as 16-byte stores.
//   tail_kernel    the same four stages as device functions inside ONE cooperative kernel that loops over waves
//                       of environments on the device: it renders whatever did not fit the arena in the first
//                       wave, and exits at once when everything did.
//
// Arithmetic follows DESIGN.md section 3 (N1-N9, N11) operation by operation (gx_math.cuh).
#pragma once
#include <cooperative_groups.h>
#include "gx_math.cuh"

namespace gx {

namespace cg = cooperative_groups;

constexpr int TILE = 16;            // tile edge, pixels (BASELINE.json north_star (3))
constexpr int NBUCKET = 8;          // depth buckets per tile (front-to-back order of a tile's list)
constexpr int NLB = 32;             // depth buckets of an environment's list of large records
constexpr int NCLASS = 8;           // cost classes of the raster tasks
constexpr int NARROW_EXT = 30000;   // sub-pixel extent below which every edge value near the box fits int32:
                                    // 2 * 30000 * (30000 + 16 * 256 + 256) < 2^31
constexpr int FQ_CAP = 256;         // fragment queue entries per warp
constexpr uint32_t BB_SKIP = 0xFFFFFFFFu;   // box word of a colour slot: not a record

// ------------------------------------------------------------------------------------------------
// record: 16 words = 64 bytes = uint4 x 4
// ------------------------------------------------------------------------------------------------
// narrow record (extent < NARROW_EXT: int32 edge functions):
//   w0..2   E_e at the box origin pixel (i0, j0), e = 0, 1, 2
//   w3..5   dx_e << 16 | (dy_e & 0xFFFF)
//   w6      box: i0 | j0 << 8 | (w-1) << 16 | (h-1) << 24   (frame coordinates, clamped to the frame)
//   w7      id << 1 | sub
//   w8..10  q = 1/w of vertices 0, 1, 2 (orientation-normalised)
//   w11..13 RGBA8 of vertices 0, 1, 2; the top byte of w11 holds the flags
// wide record: w0..2 X, w3..5 Y (snapped, orientation-normalised); rest as above
// colour slot (follows a record with F_FLOATCOL): w7..15 = c[vertex][channel] as float
enum { F_BIAS = 7, F_FLOATCOL = 8, F_WIDE = 16 };

// control words (device): cursors and the current wave
// (cursors and task counts exist once per phase of the occluder scheme: index 0 = single pass or occluder phase, 1 = second phase)
enum { C_WAVE_E0 = 0, C_WAVE_E1, C_GEOM_CUR, C_BIN_CUR = C_GEOM_CUR + 2, C_RAST_CUR = C_BIN_CUR + 2, C_CULL_DONE = C_RAST_CUR + 2,
       C_WAVE_ITEMS, C_SUM_U /* 64-bit: two words, even index */, C_WAVES = C_SUM_U + 2, C_MAX_U, C_BAD_ENVS, C_WAVE_ITEMS2,
       C_TASK_CNT = 16,
       C_NCTL = C_TASK_CNT + 2 * NCLASS };
static_assert(C_SUM_U % 2 == 0 && C_BAD_ENVS < C_TASK_CNT, "control word layout");

struct PipeParams {
    GxParams g;
    // environment table and K1 output
    float *env_mv;           // [N][K+1][12] model-view per slot
    uint32_t *env_idb;       // [N][K+1] first triangle id per slot
    uint4 *items;            // [N][item_stride]: (slot << 24 | batch, runs of 32 triangles to draw: occluder class |
                             //   the rest << 8, unused, unused)
    uint32_t *n_items;       // [N]
    uint32_t *item_pre;      // [N+1] exclusive prefix of n_items over the environments of the wave
    uint4 *wave_items;       // [ctl[C_WAVE_ITEMS]] the items of the wave's environments in one list, the environment in
                             //   the third word (pack_stage), which is what the geometry stage hands out
    uint4 *wave_items2;      // [ctl[C_WAVE_ITEMS2]] second phase of the occluder scheme: the items that still have a run
                             //   after the hi-Z test of every run's box (cull2_stage); second word = those runs
    uint32_t *U;             // [N] upper bound of the record slots of the environment
    int32_t item_stride;
    // wave allocation
    uint32_t *rec_base;      // [N] first arena slot of the environment's segment
    uint32_t *cnt;           // [N] slots used of the segment
    uint32_t *cntA;          // [N] the same after the occluder phase (the second phase bins and draws what came later)
    uint32_t *ctl;           // [C_NCTL]
    // arena
    uint4 *recs;             // [arena_slots][4]
    uint2 *bbs;              // [arena_slots] (box word, bits of the largest q = 1 / nearest depth)
    uint32_t *refs;          // [4 * arena_slots] a small record touches at most 2x2 tiles
    uint32_t arena_slots;
    // K3 output
    uint32_t *tile_off;      // [N][T * NBUCKET + 1] exclusive offsets into the environment's refs
    uint32_t *n_large;       // [N] large entries of the phase that was binned last
    uint32_t *tasks;         // [NCLASS][N * T] raster tasks (env * T + tile) per cost class
    int32_t tiles_x, tiles_y, T;
    float bucket_off, bucket_scale;   // bucket = clamp(int((bucket_off - log2(qmax)) * bucket_scale), 0, NBUCKET - 1)
    int32_t subcull;         // test every 32-triangle sub-cluster of a visible cluster against the frustum
    int32_t big_px;          // records wider or higher than this many pixels take the block path (1..TILE)
    int32_t hiz;             // 0 = no hi-Z rejection (verification)
    // occluder scheme (two phases of geometry / bin / raster per wave)
    int32_t occl;            // 1 = on
    float occl_area;         // a sub-cluster is an occluder if its screen box has this many pixels per triangle
    unsigned long long *keys;   // [N][T][256] tile keys between the two raster phases
    uint32_t *hizb;          // [N][H/4][W/8] bits of the largest depth per 8x4-pixel block after the occluder phase
    uint32_t *hizt;          // [N][hz_stride] the same per tile, then per 2x2 tiles, 4x4 tiles, ... up to one value for the
                             //   frame (levels above the first are zeroed before the call and built with atomicMax)
    int32_t hz_stride;
};

template <bool COOP, typename T>
__device__ __forceinline__ T ldi(const T *p) {   // load of data another stage produced: inside the cooperative
    if (COOP) return __ldcg(p);                  // kernel it was written during this launch, so not through L1 / the
    return __ldg(p);                             // read-only path
}

// ------------------------------------------------------------------------------------------------
// per-environment slot tables in shared memory (K1)
// ------------------------------------------------------------------------------------------------
struct EnvSmem {
    float *MV;            // [(K+1)*12] model-view per slot; slot 0 = static mesh (MV = V)
    uint32_t *id_base;    // [K+2] first triangle id of slot s; [K+1] = triangles in the environment
    uint32_t *cl_base;    // [K+2] first cluster-space index of slot s; [K+1] = clusters in the environment
    uint32_t *slot_cl;    // [K+1] global index of the slot's first cluster
    uint32_t *slot_nt;    // [K+1]
    uint32_t *slot_nc;    // [K+1]
};

__host__ __device__ inline size_t env_smem_bytes(int K) {
    return (size_t)(K + 1) * 48 + (size_t)(K + 2) * 8 + (size_t)(K + 1) * 12;
}

// slot tables, model-view matrices (N1, N2), exclusive scans of triangle and cluster counts over the K+1 slots;
// by the whole CTA (two barriers inside).  Mesh ids outside [0, n_dyn) (or [0, n_static) for the scene) are
// treated as empty slots and counted in C_BAD_ENVS.
__device__ __forceinline__ void env_setup(const PipeParams &PP, int env, const EnvSmem &es, int tid) {
    const GxParams &P = PP.g;
    const int K = P.K, lane = tid & 31, warp = tid >> 5;
    for (int sl = tid; sl <= K; sl += (int)blockDim.x) {
        int mesh = -1;
        bool bad = false;
        if (sl == 0) {
            mesh = P.env_scene[env];
            bad = mesh < 0 || mesh >= P.n_static;
        } else {
            const int m = P.inst_mesh[(size_t)env * K + (sl - 1)];
            bad = m >= P.n_dyn;
            if (m >= 0) mesh = P.n_static + m;
        }
        if (bad) { mesh = -1; atomicAdd(&PP.ctl[C_BAD_ENVS], 1u); }
        uint32_t nt = 0, nc = 0, cl0 = 0;
        if (mesh >= 0) {
            const GxMeshDev md = P.meshes[mesh];
            nt = md.nt; nc = md.ncluster; cl0 = md.cluster_off;
        }
        es.slot_nt[sl] = nt; es.slot_nc[sl] = nc; es.slot_cl[sl] = cl0;
        // N1: view matrix from the rigid camera-to-world pose C
        const float *C = P.cam_pose + (size_t)env * 16;
        float V[12];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
#pragma unroll
            for (int j = 0; j < 3; ++j) V[i * 4 + j] = C[j * 4 + i];
            V[i * 4 + 3] = -fmaf(C[8 + i], C[11], fmaf(C[4 + i], C[7], C[i] * C[3]));
        }
        float *MV = es.MV + sl * 12;
        if (sl == 0) {
#pragma unroll
            for (int k = 0; k < 12; ++k) MV[k] = V[k];
        } else {
            // N2: MV = V * M (top three rows of the instance transform)
            const float *M = P.inst_xform + ((size_t)env * K + (sl - 1)) * 16;
            float Mr[12];
#pragma unroll
            for (int k = 0; k < 12; ++k) Mr[k] = M[k];
#pragma unroll
            for (int i = 0; i < 3; ++i) {
#pragma unroll
                for (int j = 0; j < 3; ++j)
                    MV[i * 4 + j] = fmaf(V[i * 4 + 2], Mr[8 + j], fmaf(V[i * 4 + 1], Mr[4 + j], V[i * 4] * Mr[j]));
                MV[i * 4 + 3] = fmaf(V[i * 4 + 2], Mr[11], fmaf(V[i * 4 + 1], Mr[7], fmaf(V[i * 4], Mr[3], V[i * 4 + 3])));
            }
        }
    }
    __syncthreads();
    if (warp == 0) {   // exclusive scans of triangle and cluster counts over the K+1 slots
        uint32_t run_t = 0, run_c = 0;
        for (int s0 = 0; s0 <= K; s0 += 32) {
            const int s = s0 + lane;
            const uint32_t nt = s <= K ? es.slot_nt[s] : 0u, nc = s <= K ? es.slot_nc[s] : 0u;
            uint32_t it = nt, ic = nc;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t a = __shfl_up_sync(0xFFFFFFFFu, it, d), bq = __shfl_up_sync(0xFFFFFFFFu, ic, d);
                if (lane >= d) { it += a; ic += bq; }
            }
            if (s <= K) { es.id_base[s] = run_t + it - nt; es.cl_base[s] = run_c + ic - nc; }
            run_t += __shfl_sync(0xFFFFFFFFu, it, 31);
            run_c += __shfl_sync(0xFFFFFFFFu, ic, 31);
        }
        if (lane == 0) { es.id_base[K + 1] = run_t; es.cl_base[K + 1] = run_c; }
    }
    __syncthreads();
}

// ------------------------------------------------------------------------------------------------
// wave allocation, by one whole CTA: starting at environment e_first, as many consecutive environments as fit
// the arena get their segment (exclusive scan of U); the wave's cursors and per-environment counters are
// reset.  ctl[C_WAVE_E0 .. C_WAVE_E1) is the wave.
// ------------------------------------------------------------------------------------------------
__device__ void alloc_wave(const PipeParams &PP, uint32_t e_first) {
    __shared__ uint32_t s_wu[32], s_wi[32];
    __shared__ uint32_t s_run_u, s_run_i, s_end, s_fin_i;
    const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t N = (uint32_t)PP.g.N;
    if (tid == 0) { s_run_u = 0; s_run_i = 0; s_end = N; s_fin_i = 0; }
    __syncthreads();
    for (uint32_t c0 = e_first; c0 < N; c0 += NT) {
        const uint32_t e = c0 + tid;
        const uint32_t u = e < N ? __ldcg(&PP.U[e]) : 0u;
        const uint32_t ni = e < N && u ? __ldcg(&PP.n_items[e]) : 0u;   // (U = 0: nothing to draw)
        uint32_t iu = u, ii = ni;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t a = __shfl_up_sync(0xFFFFFFFFu, iu, d), b = __shfl_up_sync(0xFFFFFFFFu, ii, d);
            if (lane >= d) { iu += a; ii += b; }
        }
        if (lane == 31) { s_wu[warp] = iu; s_wi[warp] = ii; }
        __syncthreads();
        uint32_t bu = s_run_u, bi = s_run_i;
        for (int w = 0; w < warp; ++w) { bu += s_wu[w]; bi += s_wi[w]; }
        const uint32_t ex_u = bu + iu - u, ex_i = bi + ii - ni;
        // (the first environment of a wave always fits: the host sizes the arena for the largest possible U,
        // and cull_kernel empties an environment that would still exceed it)
        const bool fits = (unsigned long long)ex_u + u <= (unsigned long long)PP.arena_slots || e == e_first;
        if (e < N && !fits) atomicMin(&s_end, e);
        __syncthreads();
        const uint32_t end = s_end;
        if (e < end) {
            PP.rec_base[e] = ex_u;
            PP.item_pre[e] = ex_i;
            PP.cnt[e] = 0;
            PP.cntA[e] = 0;
        }
        if (e == end) s_fin_i = ex_i;
        if (tid == NT - 1) { s_run_u = ex_u + u; s_run_i = ex_i + ni; }
        __syncthreads();
        if (end < N) break;   // (uniform) the wave ends inside this chunk
    }
    if (tid == 0) {
        const uint32_t end = s_end, n_ch = end < N ? s_fin_i : s_run_i;
        PP.item_pre[end] = n_ch;
        PP.ctl[C_WAVE_ITEMS] = n_ch;
        PP.ctl[C_WAVE_ITEMS2] = 0;
        PP.ctl[C_WAVE_E0] = e_first;
        PP.ctl[C_WAVE_E1] = end;
        for (int c = 0; c < 2; ++c) { PP.ctl[C_GEOM_CUR + c] = 0; PP.ctl[C_BIN_CUR + c] = 0; PP.ctl[C_RAST_CUR + c] = 0; }
        PP.ctl[C_WAVES] += 1;
        for (int c = 0; c < 2 * NCLASS; ++c) PP.ctl[C_TASK_CNT + c] = 0;
    }
}

// ------------------------------------------------------------------------------------------------
// K1: the cull kernel.  One CTA per environment.
// ------------------------------------------------------------------------------------------------
template <int WARPS, bool STATS>
__global__ void __launch_bounds__(WARPS * 32) cull_kernel(const PipeParams PP) {
    extern __shared__ __align__(16) unsigned char smem[];
    const GxParams &P = PP.g;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NT = WARPS * 32;
    const int K = P.K;
    const int env = blockIdx.x;

    unsigned char *p = smem;
    EnvSmem es;
    es.MV = reinterpret_cast<float *>(p);          p += (size_t)(K + 1) * 48;
    es.id_base = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 2) * 4;
    es.cl_base = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 2) * 4;
    es.slot_cl = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 1) * 4;
    es.slot_nt = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 1) * 4;
    es.slot_nc = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 1) * 4;

    env_setup(PP, env, es, tid);
    {
        float *g_mv = PP.env_mv + (size_t)env * (size_t)(K + 1) * 12;
        uint32_t *g_idb = PP.env_idb + (size_t)env * (size_t)(K + 1);
        for (int k = tid; k < (K + 1) * 12; k += NT) g_mv[k] = es.MV[k];
        for (int k = tid; k <= K; k += NT) g_idb[k] = es.id_base[k];
    }
    const uint32_t n_cl = es.cl_base[K + 1];

    auto slot_of = [&](uint32_t g) {
        int lo = 0, hi = K;
        while (lo < hi) {   // largest slot whose first cluster index is <= g
            const int mid = (lo + hi + 1) >> 1;
            if (es.cl_base[mid] <= g) lo = mid; else hi = mid - 1;
        }
        return (uint32_t)lo;
    };

    unsigned st_tested = 0, st_drawn = 0;
    constexpr int CCH = 256;                                   // clusters per round
    constexpr int VB_CAP = CCH * GX_MAX_BATCH_PER_CLUSTER;     // batches of the visible clusters of a round
    __shared__ uint32_t s_vb[VB_CAP], s_vm[VB_CAP];
    __shared__ unsigned s_nvb, s_U, s_nitems;
    if (tid == 0) { s_U = 0; s_nitems = 0; }
    uint4 *env_items = PP.items + (size_t)env * (size_t)PP.item_stride;
    for (uint32_t c0 = 0; c0 < n_cl; c0 += CCH) {
        if (tid == 0) s_nvb = 0;
        __syncthreads();
        // step 1, one thread per cluster: frustum test of the cluster AABB; the batches of the survivors are
        // listed in shared memory
        for (uint32_t g = c0 + tid; g < min(c0 + (uint32_t)CCH, n_cl); g += NT) {
            const uint32_t s = slot_of(g);
            const GxClusterDev c = P.clusters[es.slot_cl[s] + (g - es.cl_base[s])];
            bool vis = true;
            if (P.cull) vis = box_in_frustum(cluster_box(c, es.MV + s * 12), P.fx, P.fy, P.znear, P.zfar);
            if (STATS) { ++st_tested; st_drawn += vis ? 1u : 0u; }
            if (vis) {
                const uint32_t nb = min(c.nbatch, (uint32_t)GX_MAX_BATCH_PER_CLUSTER);
                const uint32_t at = atomicAdd(&s_nvb, nb);
                for (uint32_t k = 0; k < nb; ++k) {
                    s_vb[at + k] = (s << 24) | (c.batch_off + k);
                    s_vm[at + k] = 0u;
                }
            }
        }
        __syncthreads();
        const unsigned nvb = s_nvb;
        // step 2 (K1b), one thread per run of 32 triangles of a listed batch: its AABB against the frustum, and
        // its class in the occluder scheme (bit r = occluder, bit 8 + r = the rest).  A surviving run adds its
        // triangle count to U -- four slots per triangle if its box reaches the near plane (a clipped triangle
        // leaves as up to two pieces of two slots each), one otherwise.
        for (unsigned idx = tid; idx < nvb * GX_SUBS_PER_BATCH; idx += NT) {
            const unsigned v = idx / GX_SUBS_PER_BATCH, r = idx % GX_SUBS_PER_BATCH;
            const uint32_t batch = s_vb[v] & 0xFFFFFFu, s = s_vb[v] >> 24;
            const int nt = (int)(P.batches[batch].nv_nt >> 16);
            if ((int)r * 32 >= nt) continue;
            const GxClusterDev sb = P.subs[(size_t)batch * GX_SUBS_PER_BATCH + r];
            const CamBox bx = cluster_box(sb, es.MV + s * 12);
            const bool sv = !(P.cull && PP.subcull) || box_in_frustum(bx, P.fx, P.fy, P.znear, P.zfar);
            if (sv) {
                const bool occluder = !PP.occl || sub_is_occluder(bx, P.fx, P.fy, P.W, P.H, P.znear, PP.occl_area);
                atomicOr(&s_vm[v], (occluder ? 1u : 256u) << r);
                const unsigned n = (unsigned)min(32, nt - (int)r * 32);
                atomicAdd(&s_U, (bx.wmin >= P.znear) ? n : 4u * n);
            }
        }
        __syncthreads();
        // step 3: one work item per batch that has a run left, appended to the environment's list
        for (unsigned v0 = warp * 32; v0 < nvb; v0 += NT) {
            const unsigned v = v0 + lane;
            const bool has = v < nvb && s_vm[v] != 0u;
            const unsigned m = __ballot_sync(0xFFFFFFFFu, has);
            uint32_t base = 0;
            if (lane == 0 && m) base = atomicAdd(&s_nitems, (unsigned)__popc(m));
            base = __shfl_sync(0xFFFFFFFFu, base, 0);
            if (has) env_items[base + __popc(m & ((1u << lane) - 1u))] = make_uint4(s_vb[v], s_vm[v], 0u, 0u);
        }
        __syncthreads();
    }
    __syncthreads();
    __shared__ bool s_last;
    if (tid == 0) {
        uint32_t u = s_U;
        if (u > PP.arena_slots) { u = 0; atomicAdd(&PP.ctl[C_BAD_ENVS], 1u); }   // cannot happen: see alloc_wave (the geometry
        PP.U[env] = u;                                                           // stage never sees an environment with U = 0)
        PP.n_items[env] = s_nitems;
        atomicAdd(reinterpret_cast<unsigned long long *>(&PP.ctl[C_SUM_U]), (unsigned long long)u);
        atomicMax(&PP.ctl[C_MAX_U], u);
        __threadfence();
        s_last = atomicAdd(&PP.ctl[C_CULL_DONE], 1u) == gridDim.x - 1;
    }
    if (STATS) {
#pragma unroll
        for (int d = 16; d; d >>= 1) {
            st_tested += __shfl_xor_sync(0xFFFFFFFFu, st_tested, d);
            st_drawn += __shfl_xor_sync(0xFFFFFFFFu, st_drawn, d);
        }
        if (lane == 0) {
            atomicAdd(&P.stats[GX_STAT_CLUSTERS_TESTED], (unsigned long long)st_tested);
            atomicAdd(&P.stats[GX_STAT_CLUSTERS_DRAWN], (unsigned long long)st_drawn);
        }
    }
    __syncthreads();
    if (s_last) {   // every environment's U and item count are in global memory: allocate the first wave
        __threadfence();
        alloc_wave(PP, 0u);
    }
}


// ------------------------------------------------------------------------------------------------
// K2: geometry
// ------------------------------------------------------------------------------------------------
struct GeomWarpSmem {
    int2 *vXY;            // [GX_VCAP] snapped position, X = X_OUT if behind the near plane
    float *vQ;            // [GX_VCAP] 1/w
    uint32_t *vC;         // [GX_VCAP] RGBA8
    unsigned char *lst;   // [256] batch-local triangle indices: narrow survivors from the front, slow-path
                          //       triangles (wide, or straddling the near plane) from the back
};
constexpr int GEOM_WARP_SMEM = GX_VCAP * 16 + 256;

// N6 set-up of a narrow triangle: orientation normalisation, edge values at the box origin, packed deltas and
// the top-left bias bits.  Returns false for zero area.  `swapped` tells the caller to swap attributes 1, 2.
__device__ __forceinline__ bool narrow_setup(int X[3], int Y[3], float q[3], int i0, int j0, uint32_t E0[3], uint32_t D[3],
                                             uint32_t &bias_bits, bool &swapped) {
    int A = (X[1] - X[0]) * (Y[2] - Y[0]) - (Y[1] - Y[0]) * (X[2] - X[0]);   // < 2^31: narrow
    swapped = A < 0;
    if (A == 0) return false;
    if (swapped) {
        int ti = X[1]; X[1] = X[2]; X[2] = ti;
        ti = Y[1]; Y[1] = Y[2]; Y[2] = ti;
        const float tf = q[1]; q[1] = q[2]; q[2] = tf;
    }
    const int px0 = (i0 << 8) + 128, py0 = (j0 << 8) + 128;
    bias_bits = 0;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        const int va = (e + 1) % 3, vb = (e + 2) % 3;
        const int dx = X[vb] - X[va], dy = Y[vb] - Y[va];
        const bool tl = (dy < 0) || (dy == 0 && dx > 0);
        E0[e] = (uint32_t)(dx * (py0 - Y[va]) - dy * (px0 - X[va]));
        D[e] = ((uint32_t)dx << 16) | ((uint32_t)dy & 0xFFFFu);
        bias_bits |= (tl ? 0u : 1u) << e;
    }
    return true;
}

// One record: 64 bytes at slot `at` of the arena (128 with the colour slot of a near-clipped piece) and the (box,
// qmax) word of the side array; bit 31 of the second word marks a record of the large path (box of big_px pixels
// or more, or int64 edge functions).
constexpr uint32_t BB_LARGE = 0x80000000u;
__device__ __forceinline__ void store_record(const PipeParams &PP, size_t at, bool large, bool pair, const uint32_t w[14],
                                             const float (*oc)[3], uint32_t qmax_bits) {
    uint4 *dst = PP.recs + at * 4;
    dst[0] = make_uint4(w[0], w[1], w[2], w[3]);
    dst[1] = make_uint4(w[4], w[5], w[6], w[7]);
    dst[2] = make_uint4(w[8], w[9], w[10], w[11]);
    dst[3] = make_uint4(w[12], w[13], 0u, 0u);
    PP.bbs[at] = make_uint2(w[6], qmax_bits | (large ? BB_LARGE : 0u));
    if (pair) {
        dst[4] = make_uint4(0u, 0u, 0u, 0u);
        dst[5] = make_uint4(0u, 0u, 0u, __float_as_uint(oc[0][0]));
        dst[6] = make_uint4(__float_as_uint(oc[0][1]), __float_as_uint(oc[0][2]), __float_as_uint(oc[1][0]), __float_as_uint(oc[1][1]));
        dst[7] = make_uint4(__float_as_uint(oc[1][2]), __float_as_uint(oc[2][0]), __float_as_uint(oc[2][1]), __float_as_uint(oc[2][2]));
        PP.bbs[at + 1] = make_uint2(BB_SKIP, 0u);
    }
}

// One record per lane at most (kind 0 = none, 1 = small, 2 = large; pair = a colour slot follows): the warp
// reserves its slots with one atomic.  (Slots used <= U by construction of U, cull_kernel.)
template <bool STATS>
__device__ __forceinline__ void emit_records(const PipeParams &PP, int env, uint32_t base, uint32_t U, int lane, int kind,
                                             bool pair, const uint32_t w[14], const float (*oc)[3], uint32_t qmax_bits) {
    const unsigned FULL = 0xFFFFFFFFu, lt = (1u << lane) - 1u;
    const unsigned m = __ballot_sync(FULL, kind != 0), mp = __ballot_sync(FULL, pair);
    if (m == 0u) return;
    uint32_t bs = 0;
    if (lane == 0) bs = atomicAdd(&PP.cnt[env], (unsigned)(__popc(m) + __popc(m & mp)));
    bs = __shfl_sync(FULL, bs, 0);
    if (kind == 0) return;
    const uint32_t slot = bs + (uint32_t)(__popc(m & lt) + __popc(m & mp & lt));
    if (STATS && slot + (pair ? 1u : 0u) >= U) atomicAdd(&PP.g.stats[GX_STAT_VIOLATIONS], 1ull);   // (own bounds check)
    store_record(PP, (size_t)base + slot, kind == 2, pair, w, oc, qmax_bits);
}

// K2 for one batch, by one warp.  sub_mask: bit r set = pass r of the triangle loop (32 consecutive triangles,
// one sub-cluster) is drawn; [v_lo, v_hi]: the vertices those passes reference (K1b, cull_kernel).
// hzb: in the second phase of the occluder scheme, the environment's per-block hi-Z values of the first phase: a
// triangle whose nearest vertex is behind every block its pixel box touches is dropped before set-up.
template <bool COOP, bool STATS>
__device__ __forceinline__ void geom_batch(const PipeParams &PP, const Proj &pj, uint32_t batch, const float *MV,
                                           uint32_t slot_id_base, const GeomWarpSmem &ws, int env, uint32_t base, uint32_t U,
                                           int lane, unsigned sub_mask, int v_lo, int v_hi, const uint32_t *hzb,
                                           unsigned &n_in, unsigned &n_tri, unsigned &n_hid) {
    const GxParams &P = PP.g;
    const unsigned FULL = 0xFFFFFFFFu;
    const GxBatchDev b = P.batches[batch];
    const int nt = (int)(b.nv_nt >> 16);
    float M[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) M[k] = MV[k];
    const uint32_t idb = slot_id_base + b.first_tri;
    const float4 *__restrict__ verts = P.verts + b.vert_off;
    const uchar4 *__restrict__ tris = P.tris + b.tri_off;
    const unsigned lt = (1u << lane) - 1u;

    // K2a: vertex transform, projection, snap -> warp-private staging
    for (int v = v_lo + lane; v <= v_hi; v += 32) {
        const float4 p = __ldg(&verts[v]);
        const CamVert cv = xform(M, p.x, p.y, p.z);
        int X = X_OUT, Y = 0;
        float q = 0.0f;
        if (cv.w >= P.znear) project(pj, cv.xc, cv.yc, cv.w, X, Y, q);
        ws.vXY[v] = make_int2(X, Y);
        ws.vQ[v] = q;
        ws.vC[v] = __float_as_uint(p.w);
    }
    __syncwarp();

    // K2b: near classification and pixel-centre bounding-box reject; compact narrow survivors to the front
    // of lst and slow-path triangles (wide, or straddling the near plane) to the back
    int nsurv = 0, nslow = 0;
    for (unsigned rm = sub_mask; rm; rm &= rm - 1u) {
        const int t0 = (__ffs((int)rm) - 1) << 5;
        if (t0 >= nt) break;
        const int t = t0 + lane;
        if (STATS) n_in += (lane == 0) ? (unsigned)min(32, nt - t0) : 0u;
        bool ok = false, slow = false;
        if (t < nt) {
            const uchar4 ix = __ldg(&tris[t]);
            const int2 a = ws.vXY[ix.x], bb = ws.vXY[ix.y], c = ws.vXY[ix.z];
            const int nout = (int)(a.x == X_OUT) + (int)(bb.x == X_OUT) + (int)(c.x == X_OUT);
            if (nout == 0) {
                const int Xmin = min(a.x, min(bb.x, c.x)), Xmax = max(a.x, max(bb.x, c.x));
                const int Ymin = min(a.y, min(bb.y, c.y)), Ymax = max(a.y, max(bb.y, c.y));
                const int i0 = max((Xmin + 127) >> 8, 0), i1 = min((Xmax - 128) >> 8, P.W - 1);
                const int j0 = max((Ymin + 127) >> 8, 0), j1 = min((Ymax - 128) >> 8, P.H - 1);
                if (i0 <= i1 && j0 <= j1) {
                    ok = max(Xmax - Xmin, Ymax - Ymin) < NARROW_EXT;
                    slow = !ok;
                    if (hzb && i1 - i0 < 32 && j1 - j0 < 16) {   // (at most 5 x 5 blocks)
                        uint32_t zb = 0;
                        const int bw = P.W >> 3;
                        for (int by = j0 >> 2; by <= (j1 >> 2); ++by)
                            for (int bx = i0 >> 3; bx <= (i1 >> 3); ++bx) zb = max(zb, ldi<COOP>(&hzb[by * bw + bx]));
                        const float qmax = fmaxf(ws.vQ[ix.x], fmaxf(ws.vQ[ix.y], ws.vQ[ix.z]));
                        // every depth of the triangle is >= 1/qmax (N7, up to a few ulp): hidden iff behind with margin
                        if (qmax * __uint_as_float(zb) < 1.0f - 1e-5f) { ok = false; slow = false; if (STATS) ++n_hid; }
                    }
                }
            } else if (nout < 3) {
                slow = true;
            }
        }
        const unsigned mo = __ballot_sync(FULL, ok), mc = __ballot_sync(FULL, slow);
        if (ok) ws.lst[nsurv + __popc(mo & lt)] = (unsigned char)t;
        if (slow) ws.lst[255 - (nslow + __popc(mc & lt))] = (unsigned char)t;
        nsurv += __popc(mo);
        nslow += __popc(mc);
    }
    __syncwarp();

    // K2c: set-up of the narrow survivors, 32 at a time.  Their slots are reserved with one atomic for the batch;
    // what zero-area triangles leave unused is marked as skipped.
    uint32_t bs0 = 0;
    if (lane == 0 && nsurv) bs0 = atomicAdd(&PP.cnt[env], (unsigned)nsurv);
    bs0 = __shfl_sync(FULL, bs0, 0);
    int used = 0;
    for (int g0 = 0; g0 < nsurv; g0 += 32) {
        const bool have = g0 + lane < nsurv;
        uint32_t w[14];
        uint32_t qmax_bits = 0;
        int kind = 0;
        if (have) {
            const int t = ws.lst[g0 + lane];
            const uchar4 ix = __ldg(&tris[t]);
            const int2 a = ws.vXY[ix.x], bq = ws.vXY[ix.y], c = ws.vXY[ix.z];
            int X[3] = {a.x, bq.x, c.x}, Y[3] = {a.y, bq.y, c.y};
            float q[3] = {ws.vQ[ix.x], ws.vQ[ix.y], ws.vQ[ix.z]};
            uint32_t col[3] = {ws.vC[ix.x], ws.vC[ix.y], ws.vC[ix.z]};
            int i0, i1, j0, j1;
            pixel_bbox(X, Y, P.W, P.H, i0, i1, j0, j1);   // non-empty: the triangle passed K2b
            bool swapped;
            uint32_t bias;
            const bool good = narrow_setup(X, Y, q, i0, j0, &w[0], &w[3], bias, swapped);   // zero area: dropped
            if (good) {
                if (swapped) { const uint32_t tc = col[1]; col[1] = col[2]; col[2] = tc; }
                w[6] = (uint32_t)i0 | ((uint32_t)j0 << 8) | ((uint32_t)(i1 - i0) << 16) | ((uint32_t)(j1 - j0) << 24);
                w[7] = (idb + (uint32_t)t) << 1;
                w[8] = __float_as_uint(q[0]); w[9] = __float_as_uint(q[1]); w[10] = __float_as_uint(q[2]);
                w[11] = (col[0] & 0xFFFFFFu) | (bias << 24);
                w[12] = col[1]; w[13] = col[2];
                qmax_bits = __float_as_uint(fmaxf(q[0], fmaxf(q[1], q[2])));
                kind = (i1 - i0 < PP.big_px && j1 - j0 < PP.big_px) ? 1 : 2;
                if (STATS) ++n_tri;
            }
        }
        const unsigned mg = __ballot_sync(FULL, kind != 0);
        if (STATS && kind && bs0 + (uint32_t)(used + __popc(mg & lt)) >= U) atomicAdd(&P.stats[GX_STAT_VIOLATIONS], 1ull);   // (own bounds check)
        if (kind) store_record(PP, (size_t)base + bs0 + (uint32_t)(used + __popc(mg & lt)), kind == 2, false, w, nullptr, qmax_bits);
        used += __popc(mg);
    }
    for (int k = used + lane; k < nsurv; k += 32) PP.bbs[(size_t)base + bs0 + (uint32_t)k] = make_uint2(BB_SKIP, 0u);

    // slow path: wide triangles and near-plane straddlers (N4), piece by piece
    for (int g = 0; g < nslow; g += 32) {
        const bool have = g + lane < nslow;
        CamVert cv[3];
        float c[3][3];
        uint32_t col8[3] = {0u, 0u, 0u};
        int t = 0;
        if (have) {
            t = ws.lst[255 - (g + lane)];
            const uchar4 ix = __ldg(&tris[t]);
            const float4 p0 = __ldg(&verts[ix.x]), p1 = __ldg(&verts[ix.y]), p2 = __ldg(&verts[ix.z]);
            cv[0] = xform(M, p0.x, p0.y, p0.z);
            cv[1] = xform(M, p1.x, p1.y, p1.z);
            cv[2] = xform(M, p2.x, p2.y, p2.z);
            col8[0] = __float_as_uint(p0.w); col8[1] = __float_as_uint(p1.w); col8[2] = __float_as_uint(p2.w);
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                c[0][ch] = (float)((col8[0] >> (8 * ch)) & 0xFFu);
                c[1][ch] = (float)((col8[1] >> (8 * ch)) & 0xFFu);
                c[2][ch] = (float)((col8[2] >> (8 * ch)) & 0xFFu);
            }
        }
#pragma unroll 1
        for (int sub = 0; sub < 2; ++sub) {
            Tri tri;
            float oc[3][3];
            uint32_t w[14];
            uint32_t qmax_bits = 0;
            int kind = 0;
            bool pair = false;
            if (have) {
                CamVert o[3];
                const int n_in = (int)(cv[0].w >= P.znear) + (int)(cv[1].w >= P.znear) + (int)(cv[2].w >= P.znear);
                const int np = clip_near<true>(cv, c, P.znear, sub, o, oc);
                if (sub < np) {
#pragma unroll
                    for (int k = 0; k < 3; ++k) project(pj, o[k].xc, o[k].yc, o[k].w, tri.X[k], tri.Y[k], tri.q[k]);
                    tri.id2 = ((idb + (uint32_t)t) << 1) | (unsigned)sub;
                    int i0, i1, j0, j1;
                    if (pixel_bbox(tri.X, tri.Y, P.W, P.H, i0, i1, j0, j1)) {
                        const long long A = area2(tri);
                        if (A != 0) {
                            const int ext = max(max(tri.X[0], max(tri.X[1], tri.X[2])) - min(tri.X[0], min(tri.X[1], tri.X[2])),
                                                max(tri.Y[0], max(tri.Y[1], tri.Y[2])) - min(tri.Y[0], min(tri.Y[1], tri.Y[2])));
                            const bool narrow = ext < NARROW_EXT;
                            pair = n_in < 3;       // clipped: colours were interpolated, they travel as floats
                            uint32_t cc[3] = {col8[0], col8[1], col8[2]};
                            if (A < 0) {
                                swap12(tri);
#pragma unroll
                                for (int ch = 0; ch < 3; ++ch) { const float f = oc[1][ch]; oc[1][ch] = oc[2][ch]; oc[2][ch] = f; }
                                const uint32_t tc = cc[1]; cc[1] = cc[2]; cc[2] = tc;
                            }
                            uint32_t flags = pair ? (uint32_t)F_FLOATCOL : 0u;
                            if (narrow) {
                                bool swapped;
                                uint32_t bias;
                                narrow_setup(tri.X, tri.Y, tri.q, i0, j0, &w[0], &w[3], bias, swapped);   // already normalised: no swap
                                flags |= bias;
                            } else {
                                w[0] = (uint32_t)tri.X[0]; w[1] = (uint32_t)tri.X[1]; w[2] = (uint32_t)tri.X[2];
                                w[3] = (uint32_t)tri.Y[0]; w[4] = (uint32_t)tri.Y[1]; w[5] = (uint32_t)tri.Y[2];
                                flags |= (uint32_t)F_WIDE;
                            }
                            w[6] = (uint32_t)i0 | ((uint32_t)j0 << 8) | ((uint32_t)(i1 - i0) << 16) | ((uint32_t)(j1 - j0) << 24);
                            w[7] = tri.id2;
                            w[8] = __float_as_uint(tri.q[0]); w[9] = __float_as_uint(tri.q[1]); w[10] = __float_as_uint(tri.q[2]);
                            w[11] = (cc[0] & 0xFFFFFFu) | (flags << 24);
                            w[12] = cc[1]; w[13] = cc[2];
                            qmax_bits = __float_as_uint(fmaxf(tri.q[0], fmaxf(tri.q[1], tri.q[2])));
                            kind = (narrow && i1 - i0 < PP.big_px && j1 - j0 < PP.big_px) ? 1 : 2;
                            if (STATS) ++n_tri;
                        }
                    }
                }
            }
            emit_records<STATS>(PP, env, base, U, lane, kind, pair, w, oc, qmax_bits);
        }
    }
    __syncwarp();
}

// second phase of the occluder scheme: is the box of a run of 32 triangles behind the hi-Z tiles of the first phase?
// (a function of its own: only 8 lanes of a warp get here, and its registers stay out of the triangle loops)
template <bool COOP>
__device__ __forceinline__ bool sub_hidden(const PipeParams &PP, const GxClusterDev &sb, const float *MV, uint32_t e) {
    float M[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) M[k] = ldi<COOP>(&MV[k]);
    return box_occluded<COOP>(cluster_box(sb, M), PP.hizt + (size_t)e * (size_t)PP.hz_stride, PP.tiles_x, PP.tiles_y, PP.g.fx, PP.g.fy,
                              PP.g.W, PP.g.H, PP.g.znear);
}

// The geometry stage: every warp draws items of the call's list until it is exhausted; items of environments
// outside the current wave are skipped.  phase: 0 = every run of the item, 1 = the occluder runs, 2 = the other
// runs, after a hi-Z test of each run's box against the tiles of the occluder phase.
// No CTA-level synchronisation.  warp_smem: GEOM_WARP_SMEM bytes of shared memory private to the warp.
template <bool COOP, bool STATS, bool HZ>
__device__ __forceinline__ void geom_stage(const PipeParams &PP, unsigned char *warp_smem, int phase) {
    const GxParams &P = PP.g;
    const unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31;
    const int K = P.K;
    GeomWarpSmem ws;
    ws.vXY = reinterpret_cast<int2 *>(warp_smem);
    ws.vQ = reinterpret_cast<float *>(warp_smem + GX_VCAP * 8);
    ws.vC = reinterpret_cast<uint32_t *>(warp_smem + GX_VCAP * 12);
    ws.lst = warp_smem + GX_VCAP * 16;
    Proj pj;
    pj.fx = P.fx; pj.fy = P.fy;
    pj.hw = 128.0f * (float)P.W; pj.hh = 128.0f * (float)P.H;

    unsigned st_in = 0, st_tri = 0, st_hid = 0;
    const unsigned n_items = ldi<COOP>(&PP.ctl[phase == 2 ? C_WAVE_ITEMS2 : C_WAVE_ITEMS]);
    const uint4 *items = phase == 2 ? PP.wave_items2 : PP.wave_items;
    uint32_t *cursor = &PP.ctl[C_GEOM_CUR + (phase == 2 ? 1 : 0)];
    const size_t hzb_stride = (size_t)(P.W >> 3) * (size_t)(P.H >> 2);
    unsigned next = 0;
    if (lane == 0) next = atomicAdd(cursor, 1u);
    next = __shfl_sync(FULL, next, 0);
    while (next < n_items) {
        const unsigned g = next;
        if (lane == 0) next = atomicAdd(cursor, 1u);   // draw the following item while this one is processed
        const uint4 item = ldi<COOP>(&items[g]);
        const uint32_t e = item.z, s = item.x >> 24, batch = item.x & 0xFFFFFFu;
        {
        unsigned mask = phase == 0 ? ((item.y | (item.y >> 8)) & 255u) : (item.y & 255u);   // (phase 2: the runs cull2_stage left)
        if (mask) {
            const uint32_t U = ldi<COOP>(&PP.U[e]), rbase = ldi<COOP>(&PP.rec_base[e]);
            const float *MV = PP.env_mv + ((size_t)e * (size_t)(K + 1) + s) * 12;
            // lanes 0..7: one run each -- its vertex range
            uint32_t vlo = 0xFFFFu, vhi = 0u;
            if (lane < GX_SUBS_PER_BATCH && ((mask >> lane) & 1u)) {
                const GxClusterDev sb = P.subs[(size_t)batch * GX_SUBS_PER_BATCH + lane];
                vlo = sb.batch_off; vhi = sb.nbatch;   // (fields reused: first and last vertex the run references)
            }
            {
                vlo = __reduce_min_sync(FULL, vlo);
                vhi = __reduce_max_sync(FULL, vhi);
                geom_batch<COOP, STATS>(PP, pj, batch, MV, ldi<COOP>(&PP.env_idb[(size_t)e * (size_t)(K + 1) + s]), ws, (int)e,
                                        rbase, U, lane, mask, (int)vlo, (int)vhi,
                                        HZ ? PP.hizb + (size_t)e * hzb_stride : nullptr, st_in, st_tri, st_hid);
            }
        }
        }
        next = __shfl_sync(FULL, next, 0);
    }
    if (STATS) {
#pragma unroll
        for (int d = 16; d; d >>= 1) {
            st_tri += __shfl_xor_sync(FULL, st_tri, d);
            st_hid += __shfl_xor_sync(FULL, st_hid, d);
        }
        if (lane == 0) {
            atomicAdd(&P.stats[GX_STAT_TRIS_IN], (unsigned long long)st_in);
            atomicAdd(&P.stats[GX_STAT_TRIS_RASTER], (unsigned long long)st_tri);
            atomicAdd(&P.stats[GX_STAT_TRIS_HIDDEN], (unsigned long long)st_hid);
        }
    }
}

#ifndef GEOM_MINB
#define GEOM_MINB 4
#endif
template <int WARPS, bool STATS, bool HZ>
__global__ void __launch_bounds__(WARPS * 32, GEOM_MINB) geom_kernel(const PipeParams PP, int phase) {
    extern __shared__ __align__(16) unsigned char smem[];
    geom_stage<false, STATS, HZ>(PP, smem + (size_t)(threadIdx.x >> 5) * GEOM_WARP_SMEM, phase);
}


// ------------------------------------------------------------------------------------------------
// K3: binning.  One CTA per environment at a time.
//   small records: count -> exclusive scan -> fill into per-(tile, depth bucket) lists of record indices at the
//     bottom of the environment's reference area (exact sizes, nothing can overflow);
//   large records (bit 31 of the second word of the side array): one 16-byte entry each -- (slot | wide << 31, 64-bit mask of the cells of the frame some pixel
//     of the triangle can fall in, bits of the largest q) -- sorted front to back by a counting sort over NLB
//     depth buckets, at the top of the reference area (entry i at uint4 index U - 1 - i).  A cell is a tile
//     (frames of at most 64 tiles) or 2x2 tiles; a cell is left out when some edge function is negative at all
//     four corners of it, so a tile only looks at triangles that reach it.
//   Also files every tile as a raster task under its cost class.
// phase 0 / 1 bin everything emitted so far, phase 2 what the second geometry phase added (cntA .. cnt).
// s_cnt, s_off: T * NBUCKET words of shared memory each.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int depth_bucket(const PipeParams &PP, uint32_t qmax_bits, int nb, float scale) {
    const float v = (PP.bucket_off - __log2f(__uint_as_float(qmax_bits))) * scale;
    return min(max((int)v, 0), nb - 1);
}

// cells of the frame a large record can touch
template <bool COOP>
__device__ __forceinline__ unsigned long long large_mask(const PipeParams &PP, const uint4 *rp, uint32_t bb, bool &wide) {
    const int cshift = PP.T > 64 ? 5 : 4;                       // log2 of the cell edge in pixels
    const int cells_x = (PP.g.W + (1 << cshift) - 1) >> cshift;
    const int i0 = (int)(bb & 255u), j0 = (int)((bb >> 8) & 255u);
    const int i1 = i0 + (int)((bb >> 16) & 255u), j1 = j0 + (int)(bb >> 24);
    const uint4 u0 = ldi<COOP>(rp), u1 = ldi<COOP>(rp + 1);
    const uint32_t flags = ldi<COOP>(reinterpret_cast<const uint32_t *>(rp + 2) + 3) >> 24;
    wide = (flags & F_WIDE) != 0;
    unsigned long long m = 0;
    const int ce = (1 << cshift) - 1;
    if (!wide) {
        int sx[3], sy[3], Eo[3];
        const uint32_t E[3] = {u0.x, u0.y, u0.z}, D[3] = {u0.w, u1.x, u1.y};
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const int dx = (int)D[e] >> 16, dy = (int)(short)(D[e] & 0xFFFFu);
            sx[e] = -(dy << 8);
            sy[e] = dx << 8;
            // largest value over a cell whose first pixel is the box origin, top-left bias taken off
            Eo[e] = (int)E[e] - (int)((flags >> e) & 1u) + max(ce * sx[e], 0) + max(ce * sy[e], 0);
        }
        for (int cy = j0 >> cshift; cy <= (j1 >> cshift); ++cy)
            for (int cx = i0 >> cshift; cx <= (i1 >> cshift); ++cx) {
                // the cell's corner pixels are at most one cell edge outside the box; for cells of 32 pixels the
                // edge values could leave int32, so those are only tested against the box
                bool in = true;
                if (cshift == 4) {
                    const int ox = (cx << 4) - i0, oy = (cy << 4) - j0;
#pragma unroll
                    for (int e = 0; e < 3; ++e) in = in && (Eo[e] + ox * sx[e] + oy * sy[e] >= 0);
                }
                if (in) m |= 1ull << (cy * cells_x + cx);
            }
    } else {
        for (int cy = j0 >> cshift; cy <= (j1 >> cshift); ++cy)
            for (int cx = i0 >> cshift; cx <= (i1 >> cshift); ++cx) m |= 1ull << (cy * cells_x + cx);
    }
    return m;
}

template <bool COOP, bool STATS>
__device__ __forceinline__ void bin_stage(const PipeParams &PP, uint32_t *s_cnt, uint32_t *s_off, int phase) {
    constexpr int LCAP = 1536;   // large records listed in shared memory between the two passes
    __shared__ uint32_t s_env, s_wtot[32], s_ccnt[NCLASS], s_cbase[NCLASS], s_lcnt[NLB], s_loff[NLB], s_nl, s_llist[LCAP];
    const int tid = threadIdx.x, NT = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const int T = PP.T, NK = T * NBUCKET;     // (T <= NT in every supported frame size: thread t takes tile t)
    const int pi = phase == 2 ? 1 : 0;
    const uint32_t e0 = ldi<COOP>(&PP.ctl[C_WAVE_E0]), e1 = ldi<COOP>(&PP.ctl[C_WAVE_E1]);
    const float sc_small = PP.bucket_scale, sc_large = PP.bucket_scale * (float)NLB / (float)NBUCKET;
    for (;;) {
        __syncthreads();
        if (tid == 0) s_env = e0 + atomicAdd(&PP.ctl[C_BIN_CUR + pi], 1u);
        __syncthreads();
        const uint32_t env = s_env;
        if (env >= e1) break;
        const uint32_t ns = ldi<COOP>(&PP.cnt[env]);
        const uint32_t s_lo = phase == 2 ? ldi<COOP>(&PP.cntA[env]) : 0u;
        const uint32_t U = ldi<COOP>(&PP.U[env]);
        const size_t base = ldi<COOP>(&PP.rec_base[env]);
        const uint2 *ebb = PP.bbs + base;
        const uint4 *env_recs = PP.recs + base * 4;
        uint32_t *erefs = PP.refs + 4 * base;
        uint4 *elarge = reinterpret_cast<uint4 *>(erefs);
        // Records of the small path reference every tile their box touches: at most 2x2 tiles for boxes below 16
        // pixels, so 4 words per slot always hold them; boxes up to big_px (< 32) pixels can touch 3x3.  If the exact
        // count of a first attempt does not fit the environment's reference area, the boxes of 16 pixels and more
        // join the large records and the count is taken again (which then fits by the 2x2 argument).
        bool mid_large = false;
        uint32_t n_large = 0, run = 0, sum = 0;
        auto is_large = [&](const uint2 &b) {
            return (b.y & BB_LARGE) != 0u || (mid_large && ((b.x >> 16) & 255u) >= 16u) || (mid_large && (b.x >> 24) >= 16u);
        };
        for (int attempt = 0; attempt < 2; ++attempt) {
            for (int k = tid; k < NK; k += NT) s_cnt[k] = 0;
            if (tid < NLB) s_lcnt[tid] = 0;
            if (tid == 0) s_nl = 0;
            __syncthreads();
            // count: small records per (tile, bucket), large records per bucket
            for (uint32_t s = s_lo + tid; s < ns; s += NT) {
                const uint2 b = ldi<COOP>(&ebb[s]);
                if (b.x == BB_SKIP) continue;
                if (is_large(b)) {   // listed, so that the second pass works on them with every lane
                    atomicAdd(&s_lcnt[depth_bucket(PP, b.y & ~BB_LARGE, NLB, sc_large)], 1u);
                    const uint32_t k = atomicAdd(&s_nl, 1u);
                    if (k < (uint32_t)LCAP) s_llist[k] = s;
                    continue;
                }
                const int i0 = (int)(b.x & 255u), j0 = (int)((b.x >> 8) & 255u);
                const int i1 = i0 + (int)((b.x >> 16) & 255u), j1 = j0 + (int)(b.x >> 24);
                const int bk = depth_bucket(PP, b.y, NBUCKET, sc_small);
                for (int ty = j0 >> 4; ty <= (j1 >> 4); ++ty)
                    for (int tx = i0 >> 4; tx <= (i1 >> 4); ++tx) atomicAdd(&s_cnt[(ty * PP.tiles_x + tx) * NBUCKET + bk], 1u);
            }
            __syncthreads();
            n_large = s_nl;
            if (tid == 0) {
                uint32_t r = 0;
                for (int k = 0; k < NLB; ++k) { s_loff[k] = r; r += s_lcnt[k]; s_lcnt[k] = 0; }
            }
            // exclusive scan over (tile, bucket); thread t takes tile t's buckets
            const int t = tid;
            uint32_t v[NBUCKET];
            sum = 0;
#pragma unroll
            for (int k = 0; k < NBUCKET; ++k) { v[k] = t < T ? s_cnt[t * NBUCKET + k] : 0u; sum += v[k]; }
            uint32_t inc = sum;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t a = __shfl_up_sync(0xFFFFFFFFu, inc, d);
                if (lane >= d) inc += a;
            }
            if (lane == 31) s_wtot[warp] = inc;
            __syncthreads();
            uint32_t ex = inc - sum;
            for (int w = 0; w < warp; ++w) ex += s_wtot[w];
            run = 0;
            for (int w = 0; w < (NT >> 5); ++w) run += s_wtot[w];
            if (t < T) {
                uint32_t *g_off = PP.tile_off + (size_t)env * (size_t)(NK + 1) + (size_t)t * NBUCKET;
#pragma unroll
                for (int k = 0; k < NBUCKET; ++k) { s_off[t * NBUCKET + k] = ex; g_off[k] = ex; s_cnt[t * NBUCKET + k] = 0; ex += v[k]; }
            }
            __syncthreads();
            if ((unsigned long long)run + 4ull * n_large <= 4ull * U) break;   // (uniform) the references fit
            mid_large = true;
        }
        // every tile is a raster task, filed under its cost class: references of the tile, plus a share of the
        // large records
        if (tid < NCLASS) s_ccnt[tid] = 0;
        __syncthreads();
        uint32_t my_class = 0, my_pos = 0;
        if (tid < T) {
            const uint32_t cost = sum + (n_large >> 2) + 8u;
            my_class = (uint32_t)min(NCLASS - 1, 28 - __clz((int)cost));
            my_pos = atomicAdd(&s_ccnt[my_class], 1u);
        }
        __syncthreads();
        if (tid < NCLASS && s_ccnt[tid]) s_cbase[tid] = atomicAdd(&PP.ctl[C_TASK_CNT + pi * NCLASS + tid], s_ccnt[tid]);
        __syncthreads();
        if (tid < T) PP.tasks[(size_t)my_class * (size_t)PP.g.N * (size_t)T + s_cbase[my_class] + my_pos] = env * (uint32_t)T + (uint32_t)tid;
        if (tid == 0) {
            PP.tile_off[(size_t)env * (size_t)(NK + 1) + NK] = run;
            PP.n_large[env] = n_large;
            if (phase == 1) PP.cntA[env] = ns;
            if (STATS) {
                atomicAdd(&PP.g.stats[GX_STAT_REFS], (unsigned long long)run);
                atomicAdd(&PP.g.stats[GX_STAT_LARGE], (unsigned long long)n_large);
            }
        }
        // fill
        const bool listed = n_large <= (uint32_t)LCAP;
        auto fill_large = [&](uint32_t s, const uint2 &b) {
            const uint32_t qb = b.y & ~BB_LARGE;
            const int bk = depth_bucket(PP, qb, NLB, sc_large);
            bool wide;
            const unsigned long long m = large_mask<COOP>(PP, env_recs + (size_t)s * 4, b.x, wide);
            const uint32_t at = s_loff[bk] + atomicAdd(&s_lcnt[bk], 1u);
            if (STATS && (at >= n_large || s >= ns)) atomicAdd(&PP.g.stats[GX_STAT_VIOLATIONS], 1ull);   // (own bounds check)
            elarge[U - 1 - at] = make_uint4(s | (wide ? 0x80000000u : 0u), (uint32_t)m, (uint32_t)(m >> 32), qb);
        };
        for (uint32_t s = s_lo + tid; s < ns; s += NT) {
            const uint2 b = ldi<COOP>(&ebb[s]);
            if (b.x == BB_SKIP) continue;
            if (is_large(b)) {
                if (!listed) fill_large(s, b);
                continue;
            }
            const int i0 = (int)(b.x & 255u), j0 = (int)((b.x >> 8) & 255u);
            const int i1 = i0 + (int)((b.x >> 16) & 255u), j1 = j0 + (int)(b.x >> 24);
            const int bk = depth_bucket(PP, b.y, NBUCKET, sc_small);
            for (int ty = j0 >> 4; ty <= (j1 >> 4); ++ty)
                for (int tx = i0 >> 4; tx <= (i1 >> 4); ++tx) {
                    const int key = (ty * PP.tiles_x + tx) * NBUCKET + bk;
                    const uint32_t at = s_off[key] + atomicAdd(&s_cnt[key], 1u);
                    if (STATS && (unsigned long long)at + 4ull * n_large >= 4ull * U) atomicAdd(&PP.g.stats[GX_STAT_VIOLATIONS], 1ull);   // (own bounds check)
                    erefs[at] = s;
                }
        }
        if (listed)
            for (uint32_t k = tid; k < n_large; k += NT) {
                const uint32_t s = s_llist[k];
                fill_large(s, ldi<COOP>(&ebb[s]));
            }
    }
}

template <bool STATS>
__global__ void __launch_bounds__(512) bin_kernel(const PipeParams PP, int phase) {
    extern __shared__ __align__(16) unsigned char smem[];
    uint32_t *s_cnt = reinterpret_cast<uint32_t *>(smem);
    bin_stage<false, STATS>(PP, s_cnt, s_cnt + PP.T * NBUCKET, phase);
}

// ------------------------------------------------------------------------------------------------
// K4 + K5: raster.  A warp owns one 16x16 tile at a time.
// ------------------------------------------------------------------------------------------------
// staged record of the small path (SoA: word k of record r at rec[k*32+r]); the box is clipped to the tile
enum { R_E0 = 0, R_E1, R_E2,   // E_e at the (clipped) box origin
       R_D0, R_D1, R_D2,       // dx_e << 16 | (dy_e & 0xFFFF)
       R_Q0, R_Q1, R_Q2,       // q = 1/w of vertices 0, 1, 2
       R_FA,                   // (float)A
       R_ID,                   // id << 1 | sub
       R_BB,                   // x | y << 4 | (w-1) << 8 | (h-1) << 12 | bias bits << 16   (tile-relative)
       R_SLOT,                 // slot of the record in the environment's segment
       REC_WORDS };
// staged record of the large path (same SoA area)
enum { L_E0 = 0, L_E1, L_E2,      // E_e - bias_e at the tile's first pixel
       L_SX0, L_SX1, L_SX2,       // step of E_e per pixel in x
       L_SY0, L_SY1, L_SY2,       // ... in y
       L_Q0, L_Q1, L_Q2, L_FA, L_ID, L_SLOT,
       L_CLIP,                    // cx0 | cy0 << 4 | cx1 << 8 | cy1 << 12 | bias bits << 16: the record's box inside the tile
       LREC_WORDS };
constexpr int STAGE_WORDS = (int)LREC_WORDS > (int)REC_WORDS ? (int)LREC_WORDS : (int)REC_WORDS;

struct RastWarpSmem {
    unsigned long long *fb;   // [256] keys: depth bits << 32 | record slot; KEY_BG = background
    uint32_t *rec;            // [STAGE_WORDS * 32]
    uint32_t *fq;             // [FQ_CAP] covered fragments: r | x << 5 | y << 9 (relative to the record's clipped box)
    uint32_t *hz;             // [8] bits of the largest stored depth per 8x4-pixel block; 0xFFFFFFFF = background shows
    uint32_t *pend;           // [64] small records that passed the hi-Z test and wait for a full group
};
constexpr int RAST_WARP_SMEM = 256 * 8 + STAGE_WORDS * 32 * 4 + FQ_CAP * 4 + 8 * 4 + 64 * 4;

// key of pixel (x, y) of the tile: bit 3 of the column XORed with bit 0 of the row, so that an 8x4 block of
// 64-bit keys touches every bank exactly twice (the minimum) and 4-aligned runs of a row stay contiguous
__device__ __forceinline__ int fb_idx(int x, int y) { return y * TILE + (x ^ ((y & 1) << 3)); }

// N9 on a key the warp owns, for lanes that may hit the same pixel in the same step: smaller depth wins; at
// exactly equal depth the smaller (id << 1 | sub) wins, read from the stored slot's record (rare).
template <bool COOP>
__device__ __forceinline__ void key_min_rec(unsigned long long *slot, uint32_t dbits, uint32_t idx, uint32_t id2,
                                            const uint4 *env_recs) {
    const unsigned long long key = ((unsigned long long)dbits << 32) | idx;
    unsigned long long cur = *reinterpret_cast<volatile unsigned long long *>(slot);
    for (;;) {
        const uint32_t cd = (uint32_t)(cur >> 32);
        if (dbits > cd) return;
        if (dbits == cd) {
            const uint32_t cid2 = ldi<COOP>(reinterpret_cast<const uint32_t *>(env_recs + (size_t)(uint32_t)cur * 4) + 7);
            if (id2 >= cid2) return;
        }
        const unsigned long long old = atomicCAS(slot, cur, key);
        if (old == cur) return;
        cur = old;
    }
}

// ---- large records: pixel-parallel over the tile's eight 8x4-pixel blocks ---------------------------------
// The tile's large records are set up one per lane into the staging area (edge values at the tile's first pixel,
// steps, 1/w, the box inside the tile).  Then four records at a time, lane = (record, block): a block is rejected
// if some edge function is negative at all four corners (its largest corner value is), if it misses the record's
// box, or if the record's nearest depth is behind the block's hi-Z value.  The surviving (record, block) pairs
// are drawn one after the other, one pixel per lane; the lane owns the pixel's key, so N9 is a plain compare and
// store, and the block's hi-Z value is the warp maximum of the stored depths afterwards.
template <bool COOP>
__device__ __forceinline__ void stage_large(const RastWarpSmem &ws, const uint4 *env_recs, uint32_t slot, int pos, int x0, int y0) {
    const uint4 *rp = env_recs + (size_t)slot * 4;
    const uint4 u0 = ldi<COOP>(rp), u1 = ldi<COOP>(rp + 1), u2 = ldi<COOP>(rp + 2);
    const uint32_t flags = u2.w >> 24, bb = u1.z;
    const int i0 = (int)(bb & 255u), j0 = (int)((bb >> 8) & 255u);
    const int cx0 = max(i0, x0) - x0, cx1 = min(i0 + (int)((bb >> 16) & 255u), x0 + TILE - 1) - x0;
    const int cy0 = max(j0, y0) - y0, cy1 = min(j0 + (int)(bb >> 24), y0 + TILE - 1) - y0;
    const uint32_t E[3] = {u0.x, u0.y, u0.z}, D[3] = {u0.w, u1.x, u1.y};
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        const int dx = (int)D[e] >> 16, dy = (int)(short)(D[e] & 0xFFFFu);
        const int sx = -(dy << 8), sy = dx << 8;
        ws.rec[(L_SX0 + e) * 32 + pos] = (uint32_t)sx;
        ws.rec[(L_SY0 + e) * 32 + pos] = (uint32_t)sy;
        ws.rec[(L_E0 + e) * 32 + pos] = (uint32_t)((int)E[e] + (y0 - j0) * sy + (x0 - i0) * sx - (int)((flags >> e) & 1u));
    }
    ws.rec[L_Q0 * 32 + pos] = u2.x; ws.rec[L_Q1 * 32 + pos] = u2.y; ws.rec[L_Q2 * 32 + pos] = u2.z;
    ws.rec[L_FA * 32 + pos] = __float_as_uint((float)(int)(u0.x + u0.y + u0.z));   // E_0 + E_1 + E_2 = A at any pixel
    ws.rec[L_ID * 32 + pos] = u1.w;
    ws.rec[L_SLOT * 32 + pos] = slot;
    ws.rec[L_CLIP * 32 + pos] = (uint32_t)cx0 | ((uint32_t)cy0 << 4) | ((uint32_t)cx1 << 8) | ((uint32_t)cy1 << 12) | ((flags & (uint32_t)F_BIAS) << 16);
}

template <bool COOP, bool STATS>
__device__ __forceinline__ void draw_staged_large(const PipeParams &PP, const RastWarpSmem &ws, const uint4 *env_recs, int ns,
                                                  int lane, unsigned &n_frag, unsigned &n_blk) {
    const unsigned FULL = 0xFFFFFFFFu;
    const float zfar = PP.g.zfar;
    const int b8 = lane & 7, bxo8 = (b8 & 1) * 8, byo8 = (b8 >> 1) * 4;
    const int lx = lane & 7, ly = lane >> 3;
    for (int r0 = 0; r0 < ns; r0 += 4) {
        const int rr = r0 + (lane >> 3);
        bool rej = rr >= ns;
        if (!rej) {
            const uint32_t clip = ws.rec[L_CLIP * 32 + rr];
            const int cx0 = (int)(clip & 15u), cy0 = (int)((clip >> 4) & 15u), cx1 = (int)((clip >> 8) & 15u), cy1 = (int)((clip >> 12) & 15u);
            rej = bxo8 > cx1 || bxo8 + 7 < cx0 || byo8 > cy1 || byo8 + 3 < cy0;
            if (PP.hiz) {
                const float qm = fmaxf(__uint_as_float(ws.rec[L_Q0 * 32 + rr]), fmaxf(__uint_as_float(ws.rec[L_Q1 * 32 + rr]), __uint_as_float(ws.rec[L_Q2 * 32 + rr])));
                rej = rej || (qm * __uint_as_float(ws.hz[b8]) < 1.0f - 1e-5f);
            }
#pragma unroll
            for (int e = 0; e < 3; ++e) {
                const int sx = (int)ws.rec[(L_SX0 + e) * 32 + rr], sy = (int)ws.rec[(L_SY0 + e) * 32 + rr];
                const int mx = (int)ws.rec[(L_E0 + e) * 32 + rr] + bxo8 * sx + byo8 * sy + max(7 * sx, 0) + max(3 * sy, 0);
                rej = rej || mx < 0;
            }
        }
        unsigned live = __ballot_sync(FULL, !rej);
        int cur = -1;
        int Ep[3] = {0, 0, 0}, sx[3] = {0, 0, 0}, sy[3] = {0, 0, 0}, bias[3] = {0, 0, 0}, cx0 = 0, cy0 = 0, cx1 = 0, cy1 = 0;
        float q0 = 0.f, q1 = 0.f, q2 = 0.f, fA = 0.f, qmax = 0.f;
        uint32_t slot = 0, id2 = 0;
        while (live) {
            const int bit = __ffs((int)live) - 1;
            live &= live - 1u;
            const int rec = r0 + (bit >> 3), b = bit & 7;
            if (rec != cur) {   // (uniform)
                cur = rec;
                const uint32_t clip = ws.rec[L_CLIP * 32 + rec];
                cx0 = (int)(clip & 15u); cy0 = (int)((clip >> 4) & 15u); cx1 = (int)((clip >> 8) & 15u); cy1 = (int)((clip >> 12) & 15u);
#pragma unroll
                for (int e = 0; e < 3; ++e) {
                    sx[e] = (int)ws.rec[(L_SX0 + e) * 32 + rec];
                    sy[e] = (int)ws.rec[(L_SY0 + e) * 32 + rec];
                    Ep[e] = (int)ws.rec[(L_E0 + e) * 32 + rec] + lx * sx[e] + ly * sy[e];
                    bias[e] = (int)((clip >> (16 + e)) & 1u);
                }
                q0 = __uint_as_float(ws.rec[L_Q0 * 32 + rec]); q1 = __uint_as_float(ws.rec[L_Q1 * 32 + rec]); q2 = __uint_as_float(ws.rec[L_Q2 * 32 + rec]);
                qmax = fmaxf(q0, fmaxf(q1, q2));
                fA = __uint_as_float(ws.rec[L_FA * 32 + rec]);
                slot = ws.rec[L_SLOT * 32 + rec];
                id2 = ws.rec[L_ID * 32 + rec];
            }
            // the block's hi-Z value may have moved since the record was listed
            if (PP.hiz && qmax * __uint_as_float(ws.hz[b]) < 1.0f - 1e-5f) continue;
            const int bxo = (b & 1) * 8, byo = (b >> 1) * 4;
            const int px = bxo + lx, py = byo + ly;
            const int E0 = Ep[0] + bxo * sx[0] + byo * sy[0], E1 = Ep[1] + bxo * sx[1] + byo * sy[1],
                      E2 = Ep[2] + bxo * sx[2] + byo * sy[2];
            const bool cov = px >= cx0 && px <= cx1 && py >= cy0 && py <= cy1 && (E0 | E1 | E2) >= 0;
            unsigned long long *kp = &ws.fb[fb_idx(px, py)];
            const unsigned long long ck = *kp;
            uint32_t nd = (uint32_t)(ck >> 32);
            if (cov) {
                const float f0 = (float)(E0 + bias[0]), f1 = (float)(E1 + bias[1]), f2 = (float)(E2 + bias[2]);
                const float num = fmaf(f2, q2, fmaf(f1, q1, f0 * q0));
                const float depth = fA / num;
                if (!(depth > zfar)) {
                    const uint32_t d = __float_as_uint(depth);
                    bool win = d < nd;
                    if (d == nd) win = id2 < ldi<COOP>(reinterpret_cast<const uint32_t *>(env_recs + (size_t)(uint32_t)ck * 4) + 7);
                    if (win) { *kp = ((unsigned long long)d << 32) | slot; nd = d; }
                }
            }
            const uint32_t zb = __reduce_max_sync(FULL, nd);
            if (lane == 0) ws.hz[b] = zb;
            __syncwarp();
            if (STATS) { n_frag += cov ? 1u : 0u; n_blk += lane == 0 ? 1u : 0u; }
        }
    }
    __syncwarp();
}

// a wide record (edge functions need int64): straight from its record, block by block
template <bool COOP, bool STATS>
__device__ __noinline__ void draw_wide(const PipeParams &PP, const RastWarpSmem &ws, const uint4 *env_recs, uint32_t slot,
                                       int x0, int y0, int lane, unsigned &n_frag, unsigned &n_blk) {
    const unsigned FULL = 0xFFFFFFFFu;
    const uint4 *rp = env_recs + (size_t)slot * 4;
    const uint4 u0 = ldi<COOP>(rp), u1 = ldi<COOP>(rp + 1), u2 = ldi<COOP>(rp + 2);
    const uint32_t bb = u1.z, id2 = u1.w;
    const int i0 = (int)(bb & 255u), j0 = (int)((bb >> 8) & 255u);
    const int cx0 = max(i0, x0) - x0, cx1 = min(i0 + (int)((bb >> 16) & 255u), x0 + TILE - 1) - x0;
    const int cy0 = max(j0, y0) - y0, cy1 = min(j0 + (int)(bb >> 24), y0 + TILE - 1) - y0;
    const float zfar = PP.g.zfar;
    const int b8 = lane & 7, bxo8 = (b8 & 1) * 8, byo8 = (b8 >> 1) * 4;
    const int lx = lane & 7, ly = lane >> 3;
    Tri t;
    t.X[0] = (int)u0.x; t.X[1] = (int)u0.y; t.X[2] = (int)u0.z;
    t.Y[0] = (int)u0.w; t.Y[1] = (int)u1.x; t.Y[2] = (int)u1.y;
    t.q[0] = __uint_as_float(u2.x); t.q[1] = __uint_as_float(u2.y); t.q[2] = __uint_as_float(u2.z);
    t.id2 = id2;
    const float qmax = fmaxf(t.q[0], fmaxf(t.q[1], t.q[2]));
    bool rej = bxo8 > cx1 || bxo8 + 7 < cx0 || byo8 > cy1 || byo8 + 3 < cy0;
    if (PP.hiz) rej = rej || (qmax * __uint_as_float(ws.hz[b8]) < 1.0f - 1e-5f);
    Edges E;
    edge_setup(t, area2(t), E);   // orientation-normalised by the geometry stage: area > 0
    {
        const long long pxo = (long long)(((x0 + bxo8) << 8) + 128), pyo = (long long)(((y0 + byo8) << 8) + 128);
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const long long Eb = (long long)E.dx[e] * (pyo - E.Ya[e]) - (long long)E.dy[e] * (pxo - E.Xa[e]) - E.bias[e];
            const long long sx = -(long long)E.dy[e] * 256, sy = (long long)E.dx[e] * 256;
            const long long mx = Eb + max(7 * sx, 0ll) + max(3 * sy, 0ll);
            rej = rej || mx < 0;
        }
    }
    unsigned live = __ballot_sync(FULL, lane < 8 && !rej);
    while (live) {
        const int b = __ffs((int)live) - 1;
        live &= live - 1u;
        const int px = (b & 1) * 8 + lx, py = (b >> 1) * 4 + ly;
        float f[3], num, depth;
        const bool cov = px >= cx0 && px <= cx1 && py >= cy0 && py <= cy1 && cover_depth(E, t.q, x0 + px, y0 + py, f, num, depth);
        unsigned long long *kp = &ws.fb[fb_idx(px, py)];
        const unsigned long long ck = *kp;
        uint32_t nd = (uint32_t)(ck >> 32);
        if (cov && !(depth > zfar)) {
            const uint32_t d = __float_as_uint(depth);
            bool win = d < nd;
            if (d == nd) win = id2 < ldi<COOP>(reinterpret_cast<const uint32_t *>(env_recs + (size_t)(uint32_t)ck * 4) + 7);
            if (win) { *kp = ((unsigned long long)d << 32) | slot; nd = d; }
        }
        const uint32_t zb = __reduce_max_sync(FULL, nd);
        if (lane == 0) ws.hz[b] = zb;
        if (STATS) { n_frag += cov ? 1u : 0u; n_blk += lane == 0 ? 1u : 0u; }
    }
    __syncwarp();
}

// ---- small records: slots of 4 pixels dealt evenly to the lanes, fragment queue, dense shading -------------
// load the group's records (one per lane, by slot index) into the warp's SoA staging, boxes clipped to the tile
template <bool COOP>
__device__ __forceinline__ void load_group(const RastWarpSmem &ws, const uint4 *env_recs, uint32_t slot, bool have,
                                           int x0, int y0, int lane) {
    if (have) {
        const uint4 *rp = env_recs + (size_t)slot * 4;
        const uint4 u0 = ldi<COOP>(rp), u1 = ldi<COOP>(rp + 1), u2 = ldi<COOP>(rp + 2);
        const uint32_t bb = u1.z;
        const int i0 = (int)(bb & 255u), j0 = (int)((bb >> 8) & 255u);
        const int ci0 = max(i0, x0), cj0 = max(j0, y0);
        const int ci1 = min(i0 + (int)((bb >> 16) & 255u), x0 + TILE - 1), cj1 = min(j0 + (int)(bb >> 24), y0 + TILE - 1);
        const int di = ci0 - i0, dj = cj0 - j0;
        const uint32_t E[3] = {u0.x, u0.y, u0.z}, D[3] = {u0.w, u1.x, u1.y};
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const int dx = (int)D[e] >> 16, dy = (int)(short)(D[e] & 0xFFFFu);
            ws.rec[(R_E0 + e) * 32 + lane] = E[e] + (uint32_t)((dj * dx - di * dy) << 8);
            ws.rec[(R_D0 + e) * 32 + lane] = D[e];
        }
        ws.rec[R_BB * 32 + lane] = (uint32_t)(ci0 - x0) | ((uint32_t)(cj0 - y0) << 4) | ((uint32_t)(ci1 - ci0) << 8) |
                                   ((uint32_t)(cj1 - cj0) << 12) | (((u2.w >> 24) & (uint32_t)F_BIAS) << 16);
        ws.rec[R_ID * 32 + lane] = u1.w;
        ws.rec[(R_Q0 + 0) * 32 + lane] = u2.x;
        ws.rec[(R_Q0 + 1) * 32 + lane] = u2.y;
        ws.rec[(R_Q0 + 2) * 32 + lane] = u2.z;
        ws.rec[R_FA * 32 + lane] = __float_as_uint((float)(int)(u0.x + u0.y + u0.z));   // E_0 + E_1 + E_2 = A
        ws.rec[R_SLOT * 32 + lane] = slot;
    }
    __syncwarp();
}

// K4b: depth (N7) and resolve (N9) for the queued fragments, one per lane
template <bool COOP>
__device__ __forceinline__ void shade_queue(const RastWarpSmem &ws, int qn, float zfar, const uint4 *env_recs, int lane) {
    for (int f = lane; f < qn; f += 32) {
        const uint32_t en = ws.fq[f];
        const int r = (int)(en & 31u), a = (int)((en >> 5) & 15u), b = (int)((en >> 9) & 15u);
        const uint32_t bb = ws.rec[R_BB * 32 + r];
        const int x = (int)(bb & 15u) + a, y = (int)((bb >> 4) & 15u) + b;
        unsigned long long *slot = &ws.fb[fb_idx(x, y)];
        float q[3];
#pragma unroll
        for (int e = 0; e < 3; ++e) q[e] = __uint_as_float(ws.rec[(R_Q0 + e) * 32 + r]);
        // early z: every depth of the triangle is >= 1/max(q); behind the stored depth with margin -> cannot win
        // (the stored depth of a background pixel reads as NaN: the comparison is false)
        const float stored = __uint_as_float(reinterpret_cast<volatile uint32_t *>(slot)[1]);
        if (fmaxf(q[0], fmaxf(q[1], q[2])) * stored < 1.0f - 1e-5f) continue;
        float fe[3];
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const uint32_t d = ws.rec[(R_D0 + e) * 32 + r];
            const int dx = (int)d >> 16, dy = (int)(short)(d & 0xFFFFu);
            const int Ee = (int)ws.rec[(R_E0 + e) * 32 + r] + ((b * dx - a * dy) << 8);
            fe[e] = (float)Ee;
        }
        const float num = fmaf(fe[2], q[2], fmaf(fe[1], q[1], fe[0] * q[0]));
        const float depth = __uint_as_float(ws.rec[R_FA * 32 + r]) / num;
        if (depth > zfar) continue;
        key_min_rec<COOP>(slot, __float_as_uint(depth), ws.rec[R_SLOT * 32 + r], ws.rec[R_ID * 32 + r], env_recs);
    }
    __syncwarp();
}

// K3 (inside the tile): the clipped boxes of the group's records are cut into slots of SW pixels of one row.
// Returns the lane's exclusive prefix of slot counts (Pex, record = lane) and the group's total.
template <int SW>
__device__ __forceinline__ int group_slots(const RastWarpSmem &ws, int nrec, int lane, int &Pex, unsigned &skip) {
    const unsigned FULL = 0xFFFFFFFFu;
    int ns = 0;
    if (lane < nrec) {
        const uint32_t bb = ws.rec[R_BB * 32 + lane];
        const int w = (int)((bb >> 8) & 15u) + 1, h = (int)((bb >> 12) & 15u) + 1;
        ns = h * ((w + SW - 1) / SW);
    }
    skip = __ballot_sync(FULL, lane >= nrec);   // records without slots: the slot walk steps over them
    int inc = ns;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(FULL, inc, d);
        if (lane >= d) inc += v;
    }
    Pex = inc - ns;
    return __shfl_sync(FULL, inc, 31);
}

// K4a: coverage of the T slots of the warp's group.  The slots are dealt to the lanes in equal contiguous runs
// (a lane walks through its run, moving to the next record when one is exhausted), so that lanes stay busy
// whatever the mix of triangle sizes.  The covered pixels of one pass are appended to the fragment queue and
// shaded densely by shade_queue.
template <bool COOP, bool STATS, int SW>
__device__ __forceinline__ void raster_slots(const RastWarpSmem &ws, int Pex, unsigned skip, int T, float zfar,
                                             const uint4 *env_recs, int lane, unsigned &n_frag) {
    const unsigned FULL = 0xFFFFFFFFu;
    const unsigned lt = (1u << lane) - 1u;
    const int per = (T + 31) >> 5;
    const int s0 = lane * per;
    const int n = max(0, min(per, T - s0));
    int r = 0;   // largest record index with Pex[r] <= s0
#pragma unroll
    for (int step = 16; step; step >>= 1) {
        const int cand = r + step;
        const int pc = __shfl_sync(FULL, Pex, cand);
        if (pc <= s0) r = cand;
    }
    const int off = s0 - __shfl_sync(FULL, Pex, r);

    int E0[3], dx[3], dy[3], w = 1, h = 1, cw = 1;
    auto load_rec = [&](int rr) {   // E0 := E_e - bias_e at the origin pixel, so that "covered" is all E0 >= 0
        const uint32_t bb = ws.rec[R_BB * 32 + rr];
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            E0[e] = (int)ws.rec[(R_E0 + e) * 32 + rr] - (int)((bb >> (16 + e)) & 1u);
            const uint32_t d = ws.rec[(R_D0 + e) * 32 + rr];
            dx[e] = (int)d >> 16;
            dy[e] = (int)(short)(d & 0xFFFFu);
        }
        w = (int)((bb >> 8) & 15u) + 1;
        h = (int)((bb >> 12) & 15u) + 1;
        cw = (w + SW - 1) / SW;
    };
    load_rec(r);
    int row = off / cw, chunk = off - row * cw;
    int qn = 0;
    const uint32_t fq_addr = (uint32_t)__cvta_generic_to_shared(ws.fq);
    for (int it = 0; it < per; ++it) {
        const bool act = it < n;
        const int a = chunk * SW;
        unsigned m4 = 0;   // coverage mask of the slot's SW pixels
        if (act) {
            int Ee[3], sx[3];
#pragma unroll
            for (int e = 0; e < 3; ++e) {
                Ee[e] = E0[e] + ((row * dx[e] - a * dy[e]) << 8);
                sx[e] = -(dy[e] << 8);
            }
#pragma unroll
            for (int k = 0; k < SW; ++k) {   // covered iff no edge value (bias already subtracted) is negative
                m4 |= ((unsigned)~(Ee[0] | Ee[1] | Ee[2]) >> 31) << k;
                Ee[0] += sx[0]; Ee[1] += sx[1]; Ee[2] += sx[2];
            }
            m4 &= (1u << min(SW, w - a)) - 1u;   // pixels beyond the box
        }
        // append the covered pixels: the lanes' counts (0..SW) are prefix-summed with one ballot per bit; the queue
        // is shaded first if this pass would not fit
        const int cnt = __popc(m4);
        const unsigned c0 = __ballot_sync(FULL, cnt & 1), c1 = __ballot_sync(FULL, cnt & 2), c2 = __ballot_sync(FULL, cnt & 4);
        const unsigned c3 = SW > 4 ? __ballot_sync(FULL, cnt & 8) : 0u;
        if (c0 | c1 | c2 | c3) {
            const int tot = __popc(c0) + 2 * __popc(c1) + 4 * __popc(c2) + 8 * __popc(c3);
            if (qn + tot > FQ_CAP) {
                __syncwarp();
                if (STATS) n_frag += (lane == 0) ? (unsigned)qn : 0u;
                shade_queue<COOP>(ws, qn, zfar, env_recs, lane);
                qn = 0;
            }
            uint32_t en = (uint32_t)r | ((uint32_t)a << 5) | ((uint32_t)row << 9);
            uint32_t addr = fq_addr + (uint32_t)(qn + __popc(c0 & lt) + 2 * __popc(c1 & lt) + 4 * __popc(c2 & lt) + 8 * __popc(c3 & lt)) * 4u;
#pragma unroll
            for (int k = 0; k < SW; ++k) {
                const uint32_t bit = (m4 >> k) & 1u;
                sts_if(addr, en, bit);
                addr += bit << 2;
                en += 32u;
            }
            qn += tot;
        }
        if (act) {
            if (++chunk == cw) {
                chunk = 0;
                if (++row == h) {
                    row = 0;
                    r = (__ffs((int)(~skip & ~((2u << r) - 1u))) - 1) & 31;   // next record that has slots
                    if (it + 1 < n) load_rec(r);
                }
            }
        }
    }
    __syncwarp();
    if (qn) {
        if (STATS) n_frag += (lane == 0) ? (unsigned)qn : 0u;
        shade_queue<COOP>(ws, qn, zfar, env_recs, lane);
    }
}

// K5a: colour (N8) and id of the winning record at frame pixel (x, y)
template <bool COOP>
__device__ __forceinline__ uint32_t resolve_rec(const uint4 *env_recs, uint32_t idx, int x, int y, bool want_rgb, uint32_t &id) {
    const uint4 *rp = env_recs + (size_t)idx * 4;
    const uint4 u1 = ldi<COOP>(rp + 1);
    id = u1.w >> 1;
    if (!want_rgb) return 0u;
    const uint4 u0 = ldi<COOP>(rp), u2 = ldi<COOP>(rp + 2);
    const uint32_t flags = u2.w >> 24;
    const float q[3] = {__uint_as_float(u2.x), __uint_as_float(u2.y), __uint_as_float(u2.z)};
    float f[3], c[3][3];
    if (!(flags & F_WIDE)) {
        const uint32_t bb = u1.z;
        const int a = x - (int)(bb & 255u), b = y - (int)((bb >> 8) & 255u);
        const uint32_t D[3] = {u0.w, u1.x, u1.y};
        const uint32_t E[3] = {u0.x, u0.y, u0.z};
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const int dx = (int)D[e] >> 16, dy = (int)(short)(D[e] & 0xFFFFu);
            f[e] = (float)((int)E[e] + ((b * dx - a * dy) << 8));
        }
    } else {
        Tri t;
        t.X[0] = (int)u0.x; t.X[1] = (int)u0.y; t.X[2] = (int)u0.z;
        t.Y[0] = (int)u0.w; t.Y[1] = (int)u1.x; t.Y[2] = (int)u1.y;
        t.q[0] = q[0]; t.q[1] = q[1]; t.q[2] = q[2];
        Edges E;
        edge_setup(t, area2(t), E);
        float num, depth;
        cover_depth(E, t.q, x, y, f, num, depth);   // covered by construction: this triangle won the pixel
    }
    if (flags & F_FLOATCOL) {
        const uint4 v1 = ldi<COOP>(rp + 5), v2 = ldi<COOP>(rp + 6), v3 = ldi<COOP>(rp + 7);
        c[0][0] = __uint_as_float(v1.w); c[0][1] = __uint_as_float(v2.x); c[0][2] = __uint_as_float(v2.y);
        c[1][0] = __uint_as_float(v2.z); c[1][1] = __uint_as_float(v2.w); c[1][2] = __uint_as_float(v3.x);
        c[2][0] = __uint_as_float(v3.y); c[2][1] = __uint_as_float(v3.z); c[2][2] = __uint_as_float(v3.w);
    } else {
        const uint4 u3 = ldi<COOP>(rp + 3);
        const uint32_t col[3] = {u2.w, u3.x, u3.y};
#pragma unroll
        for (int v = 0; v < 3; ++v)
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) c[v][ch] = (float)((col[v] >> (8 * ch)) & 0xFFu);
    }
    const float num = fmaf(f[2], q[2], fmaf(f[1], q[1], f[0] * q[0]));
    uint32_t out = 0;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
        const float g0 = q[0] * c[0][ch], g1 = q[1] * c[1][ch], g2 = q[2] * c[2][ch];
        const float cn = fmaf(f[2], g2, fmaf(f[1], g1, f[0] * g0));
        const float v = cn / num;
        out |= (uint32_t)fminf(255.0f, fmaxf(0.0f, rintf(v))) << (8 * ch);
    }
    return out;
}

// The raster stage: every warp draws tile tasks, heaviest class first, until none is left.
// phase 0: clear, draw, resolve (K5).  phase 1 (occluder phase): clear, draw, leave the tile's keys and its hi-Z
// values in global memory.  phase 2: reload the keys, draw what the second geometry phase added, resolve.
// warp_smem: RAST_WARP_SMEM bytes of shared memory private to the warp.
template <bool COOP, bool STATS, int PHASE>
__device__ __forceinline__ void raster_stage(const PipeParams &PP, unsigned char *warp_smem) {
    constexpr int phase = PHASE;
    const GxParams &P = PP.g;
    const unsigned FULL = 0xFFFFFFFFu;
#ifndef GX_SW1
#define GX_SW1 8
#endif
#ifndef GX_SW2
#define GX_SW2 4
#endif
    constexpr int SW = PHASE == 2 ? GX_SW2 : GX_SW1;   // pixels per slot of the slot walk (the occluder phase has the bigger boxes)
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const int W = P.W, npix = P.W * P.H, T = PP.T, NK = T * NBUCKET;
    const int pi = phase == 2 ? 1 : 0;
    RastWarpSmem ws;
    ws.fb = reinterpret_cast<unsigned long long *>(warp_smem);
    ws.rec = reinterpret_cast<uint32_t *>(warp_smem + 256 * 8);
    ws.fq = ws.rec + STAGE_WORDS * 32;
    ws.hz = ws.fq + FQ_CAP;
    ws.pend = ws.hz + 8;
    const bool want_rgb = P.rgb != nullptr || P.obs != nullptr;
    unsigned st_frag = 0, st_culled = 0, st_blk = 0, st_ldraw = 0;
    const int cshift = T > 64 ? 1 : 0;                      // a cell of the large records' masks is 1 or 2x2 tiles
    const int cells_x = (PP.tiles_x + cshift) >> cshift;
    const int hzb_w = W >> 3;

    // class list boundaries: tasks are drawn from the heaviest class down
    uint32_t cnt_c = 0;
    if (lane < NCLASS) cnt_c = ldi<COOP>(&PP.ctl[C_TASK_CNT + pi * NCLASS + (NCLASS - 1 - lane)]);   // lane l holds class NCLASS-1-l
    uint32_t inc_c = cnt_c;
#pragma unroll
    for (int d = 1; d < NCLASS; d <<= 1) {
        const uint32_t v = __shfl_up_sync(FULL, inc_c, d);
        if (lane >= d) inc_c += v;
    }
    const uint32_t n_tasks = __shfl_sync(FULL, inc_c, NCLASS - 1);
    const size_t class_cap = (size_t)P.N * (size_t)T;

    for (;;) {
        uint32_t k = 0;
        if (lane == 0) k = atomicAdd(&PP.ctl[C_RAST_CUR + pi], 1u);
        k = __shfl_sync(FULL, k, 0);
        if (k >= n_tasks) break;
        // class of task k: first lane whose inclusive prefix exceeds k
        const unsigned mc = __ballot_sync(FULL, lane < NCLASS && inc_c > k);
        const int cl = __ffs((int)mc) - 1;
        const uint32_t before = __shfl_sync(FULL, inc_c - cnt_c, cl);
        const uint32_t task = ldi<COOP>(&PP.tasks[(size_t)(NCLASS - 1 - cl) * class_cap + (k - before)]);
        const uint32_t env = task / (uint32_t)T, tile = task - env * (uint32_t)T;
        const int tx = (int)tile % PP.tiles_x, ty = (int)tile / PP.tiles_x;
        const int x0 = tx * TILE, y0 = ty * TILE;
        const size_t base = ldi<COOP>(&PP.rec_base[env]);
        const uint4 *env_recs = PP.recs + base * 4;
        const uint2 *ebb = PP.bbs + base;
        const uint32_t *erefs = PP.refs + 4 * base;
        const uint4 *elarge = reinterpret_cast<const uint4 *>(erefs);
        const uint32_t U = ldi<COOP>(&PP.U[env]), nl = ldi<COOP>(&PP.n_large[env]);
        uint4 *gkeys = reinterpret_cast<uint4 *>(PP.keys + (size_t)task * 256);
        uint32_t *ghzb = PP.hizb + (size_t)env * (size_t)hzb_w * (size_t)(P.H >> 2);

        // ---- clear the tile, or take it over from the occluder phase -------------------------------------
        {
            uint4 *f4 = reinterpret_cast<uint4 *>(ws.fb);
            if (phase == 2) {
#pragma unroll
                for (int i = 0; i < 4; ++i) f4[i * 32 + lane] = __ldcg(&gkeys[i * 32 + lane]);
                if (lane < 8) ws.hz[lane] = __ldcg(&ghzb[(ty * 4 + (lane >> 1)) * hzb_w + tx * 2 + (lane & 1)]);
            } else {
                const uint4 ones = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
#pragma unroll
                for (int i = 0; i < 4; ++i) f4[i * 32 + lane] = ones;
                if (lane < 8) ws.hz[lane] = 0xFFFFFFFFu;
            }
        }
        __syncwarp();

        // ---- large records of the environment, front to back: those whose mask has this tile's cell ----------
        {
            const int cell = (ty >> cshift) * cells_x + (tx >> cshift);
            for (uint32_t c0 = 0; c0 < nl; c0 += 32) {
                bool ov = false;
                uint4 en = make_uint4(0u, 0u, 0u, 0u);
                if (c0 + lane < nl) {
                    en = ldi<COOP>(&elarge[U - 1 - (c0 + lane)]);
                    ov = (((cell < 32 ? en.y : en.z) >> (cell & 31)) & 1u) != 0u;
                    if (ov && cshift) {   // (cells of 2x2 tiles: the record's box against this tile)
                        const uint32_t bb = ldi<COOP>(&ebb[en.x & 0x7FFFFFFFu]).x;
                        const int i0 = (int)(bb & 255u), j0 = (int)((bb >> 8) & 255u);
                        const int i1 = i0 + (int)((bb >> 16) & 255u), j1 = j0 + (int)(bb >> 24);
                        ov = i0 < x0 + TILE && i1 >= x0 && j0 < y0 + TILE && j1 >= y0;
                    }
                    if (ov && PP.hiz) {   // behind everything drawn so far in every block of the tile?
                        uint32_t tz = 0;
#pragma unroll
                        for (int i = 0; i < 8; ++i) tz = max(tz, ws.hz[i]);
                        ov = !(__uint_as_float(en.w) * __uint_as_float(tz) < 1.0f - 1e-5f);
                        if (STATS && !ov) ++st_culled;
                    }
                }
                const unsigned mw = __ballot_sync(FULL, ov && (en.x >> 31));
                const unsigned mn = __ballot_sync(FULL, ov && !(en.x >> 31));
                if (mn) {
                    if (ov && !(en.x >> 31)) stage_large<COOP>(ws, env_recs, en.x, __popc(mn & lt), x0, y0);
                    __syncwarp();
                    if (STATS) st_ldraw += lane == 0 ? (unsigned)__popc(mn) : 0u;
                    draw_staged_large<COOP, STATS>(PP, ws, env_recs, __popc(mn), lane, st_frag, st_blk);
                }
                unsigned m = mw;
                while (m) {
                    const int src = __ffs((int)m) - 1;
                    m &= m - 1u;
                    if (STATS) st_ldraw += lane == 0 ? 1u : 0u;
                    draw_wide<COOP, STATS>(PP, ws, env_recs, __shfl_sync(FULL, en.x, src) & 0x7FFFFFFFu, x0, y0, lane, st_frag, st_blk);
                }
            }
        }

        // ---- small records of the tile, nearest bucket first ---------------------------------------------
        // The references are tested against the hi-Z values of the blocks their box touches before the record is
        // loaded; the survivors wait in `pend` until a full group of 32 can be drawn.
        {
            const uint32_t *toff = PP.tile_off + (size_t)env * (size_t)(NK + 1) + (size_t)tile * NBUCKET;
            const uint32_t r_begin = ldi<COOP>(&toff[0]), r_end = ldi<COOP>(&toff[NBUCKET]);
            int np = 0;
            for (uint32_t r0 = r_begin; r0 < r_end || np > 0; r0 += 32) {
                if (r0 < r_end) {
                    const bool have = r0 + lane < r_end;
                    const uint32_t slot = have ? ldi<COOP>(&erefs[r0 + lane]) : 0u;
                    bool keep = have;
                    if (STATS && have && slot >= U) { atomicAdd(&P.stats[GX_STAT_VIOLATIONS], 1ull); keep = false; }   // (own bounds check)
                    if (keep && PP.hiz) {
                        const uint2 b = ldi<COOP>(&ebb[slot]);
                        const int i0 = (int)(b.x & 255u), j0 = (int)((b.x >> 8) & 255u);
                        const int x = max(i0, x0) - x0, y = max(j0, y0) - y0;
                        const int x1 = min(i0 + (int)((b.x >> 16) & 255u), x0 + TILE - 1) - x0, y1 = min(j0 + (int)(b.x >> 24), y0 + TILE - 1) - y0;
                        uint32_t zb = 0;
                        for (int by = y >> 2; by <= (y1 >> 2); ++by)
                            for (int bx = x >> 3; bx <= (x1 >> 3); ++bx) zb = max(zb, ws.hz[by * 2 + bx]);
                        // every depth of the triangle is >= 1/qmax (N7, up to a few ulp): hidden iff 1/qmax > zmax with margin
                        keep = !(__uint_as_float(b.y) * __uint_as_float(zb) < 1.0f - 1e-5f);
                        if (STATS && !keep) ++st_culled;
                    }
                    const unsigned mk = __ballot_sync(FULL, keep);
                    if (keep) ws.pend[np + __popc(mk & lt)] = slot;
                    np += __popc(mk);
                    __syncwarp();
                    if (np < 32 && r0 + 32 < r_end) continue;
                }
                if (np == 0) break;
                const int nrec = min(np, 32);
                const bool have = lane < nrec;
                const uint32_t slot = have ? ws.pend[lane] : 0u;
                const uint32_t carry = (32 + lane < np) ? ws.pend[32 + lane] : 0u;
                __syncwarp();
                if (32 + lane < np) ws.pend[lane] = carry;
                np -= nrec;
                load_group<COOP>(ws, env_recs, slot, have, x0, y0, lane);
                int Pex;
                unsigned skip;
                const int Tn = group_slots<SW>(ws, nrec, lane, Pex, skip);
                if (Tn) raster_slots<COOP, STATS, SW>(ws, Pex, skip, Tn, P.zfar, env_recs, lane, st_frag);
                // hi-Z values follow the small records too: cheap, and dense small geometry hides a lot
                if (PP.hiz && (r0 + 32 < r_end || np > 0)) {
#pragma unroll
                    for (int b = 0; b < 8; ++b) {
                        const uint32_t d = (uint32_t)(ws.fb[fb_idx((b & 1) * 8 + (lane & 7), (b >> 1) * 4 + (lane >> 3))] >> 32);
                        const uint32_t zb = __reduce_max_sync(FULL, d);
                        if (lane == 0) ws.hz[b] = zb;
                    }
                    __syncwarp();
                }
            }
        }
        __syncwarp();

        if constexpr (PHASE == 1) {
            // ---- occluder phase: the keys and the hi-Z values go to global memory ---------------------------
            const uint4 *f4 = reinterpret_cast<const uint4 *>(ws.fb);
#pragma unroll
            for (int i = 0; i < 4; ++i) __stcg(&gkeys[i * 32 + lane], f4[i * 32 + lane]);
            uint32_t tz = 0;
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                const uint32_t d = (uint32_t)(ws.fb[fb_idx((b & 1) * 8 + (lane & 7), (b >> 1) * 4 + (lane >> 3))] >> 32);
                const uint32_t zb = __reduce_max_sync(FULL, d);
                if (lane == b) __stcg(&ghzb[(ty * 4 + (b >> 1)) * hzb_w + tx * 2 + (b & 1)], zb);
                tz = max(tz, zb);
            }
            if (lane == 0) {
                uint32_t *hp = PP.hizt + (size_t)env * (size_t)PP.hz_stride;
                __stcg(&hp[tile], tz);
                int off = T, w = PP.tiles_x, h = PP.tiles_y;
                for (int l = 1; w > 1 || h > 1; ++l) {
                    w = (w + 1) >> 1; h = (h + 1) >> 1;
                    atomicMax(&hp[off + (ty >> l) * w + (tx >> l)], tz);
                    off += w * h;
                }
            }
            __syncwarp();
        } else {

        // ---- K5: resolve the winners, write RGB / depth / id as 16-byte stores ----------------------------
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            const int row = pass * 8 + (lane >> 2), xq = (lane & 3) * 4;
            const int a = fb_idx(xq, row);          // 4-aligned columns stay contiguous under the XOR
            const uint4 *slot = reinterpret_cast<const uint4 *>(&ws.fb[a]);
            const uint4 v0 = slot[0], v1 = slot[1];
            const uint32_t idx[4] = {v0.x, v0.z, v1.x, v1.z};
            const uint32_t db[4] = {v0.y, v0.w, v1.y, v1.w};
            uint32_t col[4], id[4];
            float4 d;
            float *dp = &d.x;
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                col[m] = 0u;
                id[m] = 0xFFFFFFFFu;
                dp[m] = 0.0f;
                if (db[m] != 0xFFFFFFFFu) {
                    dp[m] = __uint_as_float(db[m]);
                    if (want_rgb || P.id) col[m] = resolve_rec<COOP>(env_recs, idx[m], x0 + xq + m, y0 + row, want_rgb, id[m]);
                }
            }
            const size_t pix = (size_t)(y0 + row) * W + (size_t)(x0 + xq);   // within the environment's image
            const size_t out = (size_t)env * npix + pix;
            if (P.depth) *reinterpret_cast<float4 *>(P.depth + out) = d;
            if (P.obs) store_obs4(P.obs + (size_t)env * 4 * npix, (size_t)npix, pix, col, dp, P.obs_dmin, P.obs_dmax, P.obs_range);
            if (P.id) *reinterpret_cast<uint4 *>(P.id + out) = make_uint4(id[0], id[1], id[2], id[3]);
            if (P.rgb) {
                // 4 pixels = 12 bytes = 3 words per lane; the 4 lanes of a tile row hold 48 bytes = three 16-byte stores
                const uint32_t w0 = (col[0] & 0xFFFFFFu) | (col[1] << 24);
                const uint32_t w1 = ((col[1] >> 8) & 0xFFFFu) | (col[2] << 16);
                const uint32_t w2 = ((col[2] >> 16) & 0xFFu) | (col[3] << 8);
                const int g = lane & 3, gb = lane & ~3;
                uint32_t o[4];
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int m = 4 * g + r;          // word of the group's 12-word stream (g < 3)
                    const int src = gb + (m / 3) % 4, wsel = m % 3;
                    const uint32_t a0 = __shfl_sync(FULL, w0, src), a1 = __shfl_sync(FULL, w1, src), a2 = __shfl_sync(FULL, w2, src);
                    o[r] = wsel == 0 ? a0 : (wsel == 1 ? a1 : a2);
                }
                if (g < 3) {
                    uint8_t *dst = P.rgb + (out - (size_t)(4 * g)) * 3 + 16 * g;
                    *reinterpret_cast<uint4 *>(dst) = make_uint4(o[0], o[1], o[2], o[3]);
                }
            }
        }
        }
        __syncwarp();
    }

    if (STATS) {
#pragma unroll
        for (int d = 16; d; d >>= 1) {
            st_frag += __shfl_xor_sync(FULL, st_frag, d);
            st_culled += __shfl_xor_sync(FULL, st_culled, d);
            st_blk += __shfl_xor_sync(FULL, st_blk, d);
            st_ldraw += __shfl_xor_sync(FULL, st_ldraw, d);
        }
        if (lane == 0) {
            atomicAdd(&P.stats[GX_STAT_FRAGMENTS], (unsigned long long)st_frag);
            atomicAdd(&P.stats[GX_STAT_RECORDS_OCCLUDED], (unsigned long long)st_culled);
            atomicAdd(&P.stats[GX_STAT_BLOCKS_DRAWN], (unsigned long long)st_blk);
            atomicAdd(&P.stats[GX_STAT_LARGE_DRAWS], (unsigned long long)st_ldraw);
        }
    }
}

// Second phase of the occluder scheme, before its geometry: one thread per (item of the wave, run of 32 triangles):
// the box of every run that was not an occluder is tested against the hi-Z pyramid the first raster phase left
// (sub_hidden); items that keep a run are appended, with those runs as their mask, to the second item list.  Dense
// (all lanes busy, 8 per item), so that the geometry stage never sees what is hidden.
template <bool COOP, bool STATS>
__device__ __forceinline__ void cull2_stage(const PipeParams &PP) {
    __shared__ unsigned s_cnt, s_base;
    const GxParams &P = PP.g;
    const unsigned FULL = 0xFFFFFFFFu;
    const int tid = threadIdx.x, lane = tid & 31, r = lane & 7, sub = lane >> 3;
    const int K = P.K;
    const unsigned n_items = ldi<COOP>(&PP.ctl[C_WAVE_ITEMS]);
    const unsigned per_cta = blockDim.x >> 3;                           // items per CTA and round (8 threads each)
    unsigned st_hid = 0;
    for (unsigned g0 = blockIdx.x * per_cta; g0 < n_items; g0 += gridDim.x * per_cta) {   // (uniform per CTA)
        const unsigned g = g0 + (tid >> 3);
        uint4 item = make_uint4(0u, 0u, 0u, 0u);
        bool keep = false;
        if (g < n_items) {
            item = ldi<COOP>(&PP.wave_items[g]);
            if ((item.y >> (8 + r)) & 1u) {
                const uint32_t batch = item.x & 0xFFFFFFu, s = item.x >> 24, e = item.z;
                const GxClusterDev sb = P.subs[(size_t)batch * GX_SUBS_PER_BATCH + r];
                keep = !PP.hiz || !sub_hidden<COOP>(PP, sb, PP.env_mv + ((size_t)e * (size_t)(K + 1) + s) * 12, e);
                if (STATS && !keep) ++st_hid;
            }
        }
        const unsigned m = __ballot_sync(FULL, keep);
        const unsigned mine = (m >> (sub * 8)) & 255u;                 // the runs this lane's item keeps
        const bool lead = r == 0 && mine != 0u;
        const unsigned ml = __ballot_sync(FULL, lead);
        // one reservation per CTA and round
        if (tid == 0) s_cnt = 0;
        __syncthreads();
        unsigned wbase = 0;
        if (lane == 0 && ml) wbase = atomicAdd(&s_cnt, (unsigned)__popc(ml));
        wbase = __shfl_sync(FULL, wbase, 0);
        __syncthreads();
        if (tid == 0 && s_cnt) s_base = atomicAdd(&PP.ctl[C_WAVE_ITEMS2], s_cnt);
        __syncthreads();
        if (lead) PP.wave_items2[s_base + wbase + __popc(ml & ((1u << lane) - 1u))] = make_uint4(item.x, mine, item.z, 0u);
    }
    if (STATS) {
#pragma unroll
        for (int d = 16; d; d >>= 1) st_hid += __shfl_xor_sync(FULL, st_hid, d);
        if (lane == 0 && st_hid) atomicAdd(&P.stats[GX_STAT_SUBS_HIDDEN], (unsigned long long)st_hid);
    }
}

template <bool STATS>
__global__ void __launch_bounds__(256) cull2_kernel(const PipeParams PP) { cull2_stage<false, STATS>(PP); }

// The items of the wave's environments, copied into one list with the environment in the third word: the geometry
// stage then needs no search to know whose item it drew.  One warp per environment at a time.
template <bool COOP>
__device__ __forceinline__ void pack_stage(const PipeParams &PP) {
    const int lane = threadIdx.x & 31;
    const uint32_t e0 = ldi<COOP>(&PP.ctl[C_WAVE_E0]), e1 = ldi<COOP>(&PP.ctl[C_WAVE_E1]);
    const uint32_t warps = gridDim.x * (blockDim.x >> 5), w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    for (uint32_t e = e0 + w; e < e1; e += warps) {
        const uint32_t at = ldi<COOP>(&PP.item_pre[e]), n = ldi<COOP>(&PP.item_pre[e + 1]) - at;
        const uint4 *src = PP.items + (size_t)e * (size_t)PP.item_stride;
        for (uint32_t i = lane; i < n; i += 32) {
            const uint4 it = ldi<COOP>(&src[i]);
            PP.wave_items[at + i] = make_uint4(it.x, it.y, e, 0u);
        }
    }
}

__global__ void __launch_bounds__(256) pack_kernel(const PipeParams PP) { pack_stage<false>(PP); }

// the next wave, as a kernel of its own (one CTA): the host launches it, followed by the stage kernels, once for every
// wave the previous call needed, so that later waves run at full occupancy too; when no environment is left the wave
// is empty and the stage kernels that follow exit at once
__global__ void __launch_bounds__(256) wave_kernel(const PipeParams PP) {
    const uint32_t e_next = __ldcg(&PP.ctl[C_WAVE_E1]);
    if (e_next < (uint32_t)PP.g.N) {
        alloc_wave(PP, e_next);
    } else if (threadIdx.x == 0) {
        PP.ctl[C_WAVE_E0] = e_next;
        PP.ctl[C_WAVE_ITEMS] = 0;
        PP.ctl[C_WAVE_ITEMS2] = 0;
        for (int c = 0; c < 2; ++c) { PP.ctl[C_GEOM_CUR + c] = 0; PP.ctl[C_BIN_CUR + c] = 0; PP.ctl[C_RAST_CUR + c] = 0; }
        for (int c = 0; c < 2 * NCLASS; ++c) PP.ctl[C_TASK_CNT + c] = 0;
    }
}

#ifndef RAST_MINB
#define RAST_MINB 4
#endif
template <int WARPS, bool STATS, int PHASE>
__global__ void __launch_bounds__(WARPS * 32, RAST_MINB) raster_kernel(const PipeParams PP) {
    extern __shared__ __align__(16) unsigned char smem[];
    raster_stage<false, STATS, PHASE>(PP, smem + (size_t)(threadIdx.x >> 5) * RAST_WARP_SMEM);
}

// ------------------------------------------------------------------------------------------------
// The tail: ONE cooperative kernel that runs the stages wave after wave on the device until every environment
// is rendered.  After the first wave of ordinary launches it finds ctl[C_WAVE_E1] == N in the steady state and
// exits at once; when the arena was too small for the whole batch it renders the rest, as many environments per
// wave as fit, so that no input can make the path drop triangles (and none needs a second implementation).
// ------------------------------------------------------------------------------------------------
constexpr int TAIL_WARPS = 8;
__host__ __device__ inline size_t tail_smem_bytes(int T) {
    size_t a = (size_t)TAIL_WARPS * GEOM_WARP_SMEM, b = (size_t)TAIL_WARPS * RAST_WARP_SMEM, c = (size_t)2 * T * NBUCKET * 4;
    size_t m = a > b ? a : b;
    return m > c ? m : c;
}

template <bool STATS>
__global__ void __launch_bounds__(TAIL_WARPS * 32, 3) tail_kernel(const PipeParams PP) {
    extern __shared__ __align__(16) unsigned char smem[];
    cg::grid_group grid = cg::this_grid();
    const int warp = threadIdx.x >> 5;
    for (;;) {
        const uint32_t e_next = __ldcg(&PP.ctl[C_WAVE_E1]);
        if (e_next >= (uint32_t)PP.g.N) break;
        grid.sync();   // every CTA has read the end of the previous wave before it moves
        if (blockIdx.x == 0) alloc_wave(PP, e_next);
        grid.sync();
        pack_stage<true>(PP);
        grid.sync();
        for (int phase = PP.occl ? 1 : 0; phase <= (PP.occl ? 2 : 0); ++phase) {
            if (phase == 2) {
                cull2_stage<true, STATS>(PP);
                grid.sync();
            }
            if (phase == 2 && PP.hiz) geom_stage<true, STATS, true>(PP, smem + (size_t)warp * GEOM_WARP_SMEM, phase);
            else geom_stage<true, STATS, false>(PP, smem + (size_t)warp * GEOM_WARP_SMEM, phase);
            grid.sync();
            bin_stage<true, STATS>(PP, reinterpret_cast<uint32_t *>(smem), reinterpret_cast<uint32_t *>(smem) + PP.T * NBUCKET, phase);
            grid.sync();
            if (phase == 0) raster_stage<true, STATS, 0>(PP, smem + (size_t)warp * RAST_WARP_SMEM);
            else if (phase == 1) raster_stage<true, STATS, 1>(PP, smem + (size_t)warp * RAST_WARP_SMEM);
            else raster_stage<true, STATS, 2>(PP, smem + (size_t)warp * RAST_WARP_SMEM);
            grid.sync();
        }
    }
}

}  // namespace gx
