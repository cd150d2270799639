// gx_pipeline.cuh -- the render path of gx_render_batch (sm_100a): cull kernel -> work list -> geometry kernel ->
// triangle-record pool -> raster order -> raster kernel.  DESIGN.md section 5.
//
//   cull_kernel   K1: per environment, cluster AABBs against the frustum, then the 32-triangle sub-clusters of
//                 the survivors (frustum; class and hi-Z tiles in the occluder scheme); one 16-byte work item
//                 per batch that has a run of triangles left.
//   geom_kernel   K2: vertex transform / clip / snap / set-up.  No frame in shared memory and no CTA-level
//                 synchronisation, so four 8-warp CTAs fit an SM at 64 registers per thread; every triangle
//                 that survives the exact pixel-centre bounding-box test leaves as one 64-byte record per band
//                 it touches, in that (environment, band)'s segment of the record pool.
//   order_kernel  the (environment, band) raster tasks sorted by estimated cost, heaviest first.
//   raster_kernel K3 + K4 + K5.  Persistent CTAs, two per SM; a task's band of 64-bit (depth, record slot) keys
//                 lives in shared memory; warps draw groups of 32 records, cut their bounding boxes into
//                 8-pixel slots dealt evenly to the lanes, queue the covered pixels and shade them densely; the
//                 winner's colour is resolved from its record and RGB / depth (or the packed observation)
//                 leave as 16-byte stores.
// With the occluder scheme the four kernels run twice: big-triangle sub-clusters first, the rest culled against
// the hi-Z tiles the first raster pass leaves behind.
//
// An environment whose records do not fit a pool segment is flagged by the geometry kernel, skipped by the
// raster kernel and rendered by the single-kernel path of gx_kernels.cuh (render_kernel), which needs no
// pool.  Arithmetic follows DESIGN.md section 3 (N1-N9, N11) operation by operation.
#pragma once
#include "gx_kernels.cuh"

namespace gx {

// ------------------------------------------------------------------------------------------------
// record layout: 16 words = 64 bytes, one uint4 x 4
// ------------------------------------------------------------------------------------------------
// narrow record (bounding-box extent < NARROW_EXT sub-pixel units: every edge value fits int32):
//   w0..2  E_e at the bounding-box origin pixel (i0, j0), e = 0, 1, 2
//   w3..5  dx_e << 16 | (dy_e & 0xFFFF)
//   w6     i0 | j0 << 7 | (w-1) << 14 | (h-1) << 21 | bias bits << 28 | float-colour flag << 31
//   w7     id << 1 | sub
//   w8..10 q = 1/w of vertices 0, 1, 2 (orientation-normalised)
//   w11..13 RGBA8 of vertices 0, 1, 2 (unused if the float-colour flag is set)
// colour slot (follows a narrow record with the flag set, and every wide record):
//   w0..2 = -1, w3..6 = 0  (as a narrow record it covers nothing)   w7..15 = c[vertex][channel] as float
// wide record (always followed by a colour slot):
//   w0..2 X, w3..5 Y (snapped, orientation-normalised), w7 id2, w8..10 q
enum { P_E0 = 0, P_D0 = 3, P_BB = 6, P_ID = 7, P_Q0 = 8, P_C0 = 11 };
constexpr uint32_t BB_FLOATCOL = 0x80000000u;

struct PipeParams {
    GxParams g;              // N = environments of this chunk; per-call arrays already offset to the chunk
    uint4 *recs;             // [N][cap_n + cap_w][4]
    uint32_t *cnt;           // [N][2]: narrow slots, wide slots appended
    uint32_t *env_flag;      // [N]: 1 = pool segment overflowed, render with the single-kernel path
    unsigned int *counters;  // [0] geometry item counter, [1] raster env counter, [2] items in the work list
    uint4 *items;            // work list: (slot << 24 | batch, environment, mask of the 32-triangle runs to draw,
                             //            first | last << 16 vertex those runs reference)
    float *env_mv;           // [N][K+1][12] model-view per slot
    uint32_t *env_idb;       // [N][K+1] first triangle id per slot
    uint32_t *order;         // [N] raster order of the environments
    uint32_t *maxrec;        // [2] largest narrow / wide record count of any task of the call (sizes the next call's pool)
    uint32_t *cnt1;          // [N][2] record counts at the end of the occluder phase
    float *thr;              // [N] occluder phase: clusters with wmin < thr are drawn first
    float *hiz;              // [N][HZ_STRIDE] max depth per 8x8-pixel tile (stride 16) and per 32x32 tile (at +256)
    unsigned long long *frames;   // [N][W*H] frame keys between the two raster phases
    int32_t occl_pct;        // share of the frustum-visible clusters (nearest first) drawn in the occluder phase
    int32_t cap_n, cap_w;    // slots per (environment, band)
    int32_t subcull;         // geometry: test every 32-triangle sub-cluster of a batch (frustum; hi-Z in phase 2)
    int32_t phase, nphase;   // occluder scheme: pass 1 .. nphase of nphase (2 or 3); 0 = single pass
    float occl_area;         // a sub-cluster is a 'big-triangle' occluder if its screen box has this many pixels per triangle
    int32_t bands, bh;       // horizontal bands per frame, rows per band (H = bands * bh)
    int32_t big_slots, chunk_slots;   // raster pass B: groups above big_slots are drawn in chunks of chunk_slots
};

constexpr int HZ_STRIDE = 288;   // 16x16 tiles of 8x8 pixels, then 4x4 tiles of 32x32 pixels at +256

// Occlusion test of a cluster's camera-space box against the hi-Z tiles of the occluder phase: true only if
// every fragment the cluster can produce is strictly behind what is already drawn at every pixel it can
// touch (so it can never win N9), which leaves the image bit-identical (N10).
__device__ __forceinline__ bool box_occluded(const CamBox &b, const float *hz, float fx, float fy, int W, int H, float znear) {
    if (!(b.wmin >= znear)) return false;   // reaches the near plane: no screen bound
    const float xl = b.cx - b.ex, xh = b.cx + b.ex, yl = b.cy - b.ey, yh = b.cy + b.ey;
    const float iw0 = 1.0f / b.wmin, iw1 = 1.0f / b.wmax;
    const float nxl = fx * xl * (xl >= 0.0f ? iw1 : iw0), nxh = fx * xh * (xh >= 0.0f ? iw0 : iw1);
    const float nyl = fy * yl * (yl >= 0.0f ? iw1 : iw0), nyh = fy * yh * (yh >= 0.0f ? iw0 : iw1);
    // pixel range, padded by one pixel for the 1/256 snap and the float error of the box arithmetic
    const float fW = (float)W, fH = (float)H;
    const int pxl = (int)fminf(fmaxf(floorf((nxl * 0.5f + 0.5f) * fW) - 1.0f, 0.0f), fW - 1.0f);
    const int pxh = (int)fminf(fmaxf(floorf((nxh * 0.5f + 0.5f) * fW) + 1.0f, 0.0f), fW - 1.0f);
    const int pyl = (int)fminf(fmaxf(floorf((-nyh * 0.5f + 0.5f) * fH) - 1.0f, 0.0f), fH - 1.0f);
    const int pyh = (int)fminf(fmaxf(floorf((-nyl * 0.5f + 0.5f) * fH) + 1.0f, 0.0f), fH - 1.0f);
    float zmax = 0.0f;
    if (((pxh >> 3) - (pxl >> 3) + 1) * ((pyh >> 3) - (pyl >> 3) + 1) <= 16) {
        for (int ty = pyl >> 3; ty <= (pyh >> 3); ++ty)
            for (int tx = pxl >> 3; tx <= (pxh >> 3); ++tx) zmax = fmaxf(zmax, hz[ty * 16 + tx]);
    } else {
        for (int ty = pyl >> 5; ty <= (pyh >> 5); ++ty)
            for (int tx = pxl >> 5; tx <= (pxh >> 5); ++tx) zmax = fmaxf(zmax, hz[256 + ty * 4 + tx]);
    }
    return b.wmin * (1.0f - 1e-4f) > zmax;
}

// class of a sub-cluster (32 triangles) in the occluder scheme: 0 = drawn in the first pass, ..., n - 1 = in the last.
// Big-triangle sub-clusters (screen box area / 32 >= occl_area, or reaching the near plane) are the occluders:
// they cover many pixels for little geometry.  With three passes the far ones of them (wmin >= thr) wait for
// the second pass.  Any classification gives the same image; this one only decides what can be culled.
__device__ __forceinline__ int sub_class(const CamBox &b, float fx, float fy, int W, int H, float znear, float occl_area,
                                         float thr, int nphase) {
    if (!(b.wmin >= znear)) return 0;
    const float iw = 1.0f / b.wmin;   // the nearest depth gives the largest possible screen box
    const float wpx = fminf(2.0f * b.ex * fx * iw * 0.5f * (float)W, (float)W);
    const float hpx = fminf(2.0f * b.ey * fy * iw * 0.5f * (float)H, (float)H);
    const bool big = wpx * hpx >= occl_area * 32.0f;
    if (nphase == 2) return big ? 0 : 1;
    return big ? (b.wmin < thr ? 0 : 1) : 2;
}

struct GeomWarpSmem {
    int2 *vXY;            // [GX_VCAP]
    float *vQ;            // [GX_VCAP]
    uint32_t *vC;         // [GX_VCAP] RGBA8
    unsigned char *lst;   // [256]
};
constexpr int GEOM_WARP_SMEM = GX_VCAP * 16 + 256;
#ifndef GEOM_MINB
#define GEOM_MINB 4
#endif

__host__ __device__ inline size_t geom_smem_bytes(int K, int warps) {
    size_t b = (size_t)warps * GEOM_WARP_SMEM + env_smem_bytes(K);
    return (b + 15) & ~(size_t)15;
}

// N6 set-up of a narrow triangle: orientation normalisation, edge values at the bounding-box origin, packed
// deltas and the BB word.  Returns false for zero area.  `swapped` tells the caller to swap attributes 1, 2.
__device__ __forceinline__ bool narrow_setup(int X[3], int Y[3], float q[3], int i0, int i1, int j0, int j1,
                                             uint32_t E0[3], uint32_t D[3], uint32_t &bb, bool &swapped) {
    int A = (X[1] - X[0]) * (Y[2] - Y[0]) - (Y[1] - Y[0]) * (X[2] - X[0]);   // < 2^31: narrow
    swapped = A < 0;
    if (A == 0) return false;
    if (swapped) {
        int ti = X[1]; X[1] = X[2]; X[2] = ti;
        ti = Y[1]; Y[1] = Y[2]; Y[2] = ti;
        const float tf = q[1]; q[1] = q[2]; q[2] = tf;
    }
    const int px0 = (i0 << 8) + 128, py0 = (j0 << 8) + 128;
    uint32_t bias_bits = 0;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        const int va = (e + 1) % 3, vb = (e + 2) % 3;
        const int dx = X[vb] - X[va], dy = Y[vb] - Y[va];
        const bool tl = (dy < 0) || (dy == 0 && dx > 0);
        E0[e] = (uint32_t)(dx * (py0 - Y[va]) - dy * (px0 - X[va]));
        D[e] = ((uint32_t)dx << 16) | ((uint32_t)dy & 0xFFFFu);
        bias_bits |= (tl ? 0u : 1u) << e;
    }
    bb = (uint32_t)i0 | ((uint32_t)j0 << 7) | ((uint32_t)(i1 - i0) << 14) | ((uint32_t)(j1 - j0) << 21) | (bias_bits << 28);
    return true;
}

__device__ __forceinline__ void store_colour_slot(uint4 *dst, const float c[3][3], uint32_t id2) {
    dst[0] = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0u);
    dst[1] = make_uint4(0u, 0u, 0u, __float_as_uint(c[0][0]));
    dst[2] = make_uint4(__float_as_uint(c[0][1]), __float_as_uint(c[0][2]), __float_as_uint(c[1][0]), __float_as_uint(c[1][1]));
    dst[3] = make_uint4(__float_as_uint(c[1][2]), __float_as_uint(c[2][0]), __float_as_uint(c[2][1]), __float_as_uint(c[2][2]));
    (void)id2;
}

// The frame is cut into PP.bands horizontal bands of PP.bh rows; every (environment, band) pair is one raster
// task with its own record lists ("virtual environment" v = env * bands + band).  emit_narrow appends a set-up
// narrow record to the list of every band its bounding box touches, with the box clipped to the band's rows
// (edge values moved to the new origin, j0 relative to the band), so that the raster kernel needs no clipping.
// Called converged by the whole warp; PAIR: a colour slot (oc) follows the record.
template <bool PAIR>
__device__ __forceinline__ void emit_narrow(const PipeParams &PP, int env, int lane, bool valid, const uint32_t E0[3],
                                            const uint32_t D[3], uint32_t bbw, int j0, int j1, uint32_t id2,
                                            const float q[3], const uint32_t col[3], const float (*oc)[3], bool &overflow) {
    const unsigned FULL = 0xFFFFFFFFu;
    const unsigned lt = (1u << lane) - 1u;
    for (int b = 0; b < PP.bands; ++b) {
        const int lo = b * PP.bh, hi = lo + PP.bh - 1;
        const bool touch = valid && j0 <= hi && j1 >= lo;
        const unsigned m = __ballot_sync(FULL, touch);
        if (m == 0u) continue;
        const int v = env * PP.bands + b;
        const uint32_t n = (PAIR ? 2u : 1u) * (uint32_t)__popc(m);
        uint32_t base = 0;
        if (lane == 0) base = atomicAdd(&PP.cnt[2 * v], n);
        base = __shfl_sync(FULL, base, 0);
        if (base + n > (uint32_t)PP.cap_n) { overflow = true; continue; }
        if (touch) {
            const int jj0 = max(j0, lo), jj1 = min(j1, hi), dj = jj0 - j0;
            uint32_t E[3];
#pragma unroll
            for (int e = 0; e < 3; ++e) E[e] = E0[e] + (uint32_t)((dj * ((int)D[e] >> 16)) << 8);
            const uint32_t bb = (bbw & ~((127u << 7) | (127u << 21))) | ((uint32_t)(jj0 - lo) << 7) | ((uint32_t)(jj1 - jj0) << 21);
            uint4 *dst = PP.recs + ((size_t)v * (size_t)(PP.cap_n + PP.cap_w) + base + (PAIR ? 2u : 1u) * (uint32_t)__popc(m & lt)) * 4;
            dst[0] = make_uint4(E[0], E[1], E[2], D[0]);
            dst[1] = make_uint4(D[1], D[2], bb | (PAIR ? BB_FLOATCOL : 0u), id2);
            dst[2] = make_uint4(__float_as_uint(q[0]), __float_as_uint(q[1]), __float_as_uint(q[2]), PAIR ? 0u : col[0]);
            dst[3] = PAIR ? make_uint4(0u, 0u, 0u, 0u) : make_uint4(col[1], col[2], 0u, 0u);
            if (PAIR) store_colour_slot(dst + 4, oc, id2);
        }
    }
}

// wide record + colour slot, appended to the wide list of every band the (frame-clamped) rows j0..j1 touch
__device__ __forceinline__ void emit_wide(const PipeParams &PP, int env, int lane, bool valid, const Tri &tri, int j0, int j1,
                                          const float (*oc)[3], bool &overflow) {
    const unsigned FULL = 0xFFFFFFFFu;
    const unsigned lt = (1u << lane) - 1u;
    for (int b = 0; b < PP.bands; ++b) {
        const int lo = b * PP.bh, hi = lo + PP.bh - 1;
        const bool touch = valid && j0 <= hi && j1 >= lo;
        const unsigned m = __ballot_sync(FULL, touch);
        if (m == 0u) continue;
        const int v = env * PP.bands + b;
        const uint32_t n = 2u * (uint32_t)__popc(m);
        uint32_t base = 0;
        if (lane == 0) base = atomicAdd(&PP.cnt[2 * v + 1], n);
        base = __shfl_sync(FULL, base, 0);
        if (base + n > (uint32_t)PP.cap_w) { overflow = true; continue; }
        if (touch) {
            uint4 *dst = PP.recs + ((size_t)v * (size_t)(PP.cap_n + PP.cap_w) + (size_t)PP.cap_n + base + 2u * (uint32_t)__popc(m & lt)) * 4;
            dst[0] = make_uint4((uint32_t)tri.X[0], (uint32_t)tri.X[1], (uint32_t)tri.X[2], (uint32_t)tri.Y[0]);
            dst[1] = make_uint4((uint32_t)tri.Y[1], (uint32_t)tri.Y[2], 0u, tri.id2);
            dst[2] = make_uint4(__float_as_uint(tri.q[0]), __float_as_uint(tri.q[1]), __float_as_uint(tri.q[2]), 0u);
            dst[3] = make_uint4(0u, 0u, 0u, 0u);
            store_colour_slot(dst + 4, oc, tri.id2);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// geometry: K2 for one batch, by one warp.  sub_mask: bit r set = pass r of the triangle loop (32 consecutive
// triangles, one sub-cluster) is drawn; [v_lo, v_hi]: the vertices those passes reference (K1b, cull_kernel)
// ------------------------------------------------------------------------------------------------
template <bool STATS>
__device__ __forceinline__ void geom_batch(const PipeParams &PP, const Proj &pj, uint32_t batch, const float *__restrict__ MV,
                                           uint32_t slot_id_base, const GeomWarpSmem &ws, int env, int lane,
                                           unsigned sub_mask, int v_lo, int v_hi, bool &overflow, unsigned &n_in,
                                           unsigned &n_tri) {
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
    if (STATS) n_in += (lane == 0) ? 32u * (unsigned)__popc(sub_mask & ((nt + 31) / 32 < 32 ? (1u << ((nt + 31) / 32)) - 1u : 0xFFFFFFFFu)) : 0u;

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
    for (int t0 = 0; t0 < nt; t0 += 32) {
        if (!((sub_mask >> (t0 >> 5)) & 1u)) continue;
        const int t = t0 + lane;
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

    // K2c: set-up of the narrow survivors, 32 at a time; each leaves as one record per band it touches
    for (int g0 = 0; g0 < nsurv; g0 += 32) {
        const bool have = g0 + lane < nsurv;
        uint32_t E0[3] = {0u, 0u, 0u}, D[3] = {0u, 0u, 0u}, bbw = 0u, col[3] = {0u, 0u, 0u}, id2 = 0u;
        float q[3] = {0.0f, 0.0f, 0.0f};
        int j0 = 0, j1 = 0;
        bool good = false;
        if (have) {
            const int t = ws.lst[g0 + lane];
            const uchar4 ix = __ldg(&tris[t]);
            const int2 a = ws.vXY[ix.x], bq = ws.vXY[ix.y], c = ws.vXY[ix.z];
            int X[3] = {a.x, bq.x, c.x}, Y[3] = {a.y, bq.y, c.y};
            q[0] = ws.vQ[ix.x]; q[1] = ws.vQ[ix.y]; q[2] = ws.vQ[ix.z];
            col[0] = ws.vC[ix.x]; col[1] = ws.vC[ix.y]; col[2] = ws.vC[ix.z];
            int i0, i1;
            pixel_bbox(X, Y, P.W, P.H, i0, i1, j0, j1);
            bool swapped;
            good = narrow_setup(X, Y, q, i0, i1, j0, j1, E0, D, bbw, swapped);   // zero area: dropped
            if (swapped) { const uint32_t tc = col[1]; col[1] = col[2]; col[2] = tc; }
            id2 = (idb + (uint32_t)t) << 1;
            if (STATS) n_tri += good ? 1u : 0u;
        }
        emit_narrow<false>(PP, env, lane, good, E0, D, bbw, j0, j1, id2, q, col, nullptr, overflow);
    }

    // slow path: wide triangles and near-plane straddlers (N4), piece by piece
    for (int g = 0; g < nslow; g += 32) {
        const bool have = g + lane < nslow;
        CamVert cv[3];
        float c[3][3];
        int t = 0;
        if (have) {
            t = ws.lst[255 - (g + lane)];
            const uchar4 ix = __ldg(&tris[t]);
            const float4 p0 = __ldg(&verts[ix.x]), p1 = __ldg(&verts[ix.y]), p2 = __ldg(&verts[ix.z]);
            cv[0] = xform(M, p0.x, p0.y, p0.z);
            cv[1] = xform(M, p1.x, p1.y, p1.z);
            cv[2] = xform(M, p2.x, p2.y, p2.z);
            const uint32_t r0 = __float_as_uint(p0.w), r1 = __float_as_uint(p1.w), r2 = __float_as_uint(p2.w);
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                c[0][ch] = (float)((r0 >> (8 * ch)) & 0xFFu);
                c[1][ch] = (float)((r1 >> (8 * ch)) & 0xFFu);
                c[2][ch] = (float)((r2 >> (8 * ch)) & 0xFFu);
            }
        }
#pragma unroll 1
        for (int sub = 0; sub < 2; ++sub) {
            Tri tri;
            float oc[3][3];
            bool narrow = false, wide = false;
            int i0 = 0, i1 = 0, j0 = 0, j1 = 0;
            if (have) {
                CamVert o[3];
                const int np = clip_near<true>(cv, c, P.znear, sub, o, oc);
                if (sub < np) {
#pragma unroll
                    for (int k = 0; k < 3; ++k) project(pj, o[k].xc, o[k].yc, o[k].w, tri.X[k], tri.Y[k], tri.q[k]);
                    tri.id2 = ((idb + (uint32_t)t) << 1) | (unsigned)sub;
                    if (pixel_bbox(tri.X, tri.Y, P.W, P.H, i0, i1, j0, j1)) {
                        const long long A = area2(tri);
                        if (A != 0) {
                            const int ext = max(max(tri.X[0], max(tri.X[1], tri.X[2])) - min(tri.X[0], min(tri.X[1], tri.X[2])),
                                                max(tri.Y[0], max(tri.Y[1], tri.Y[2])) - min(tri.Y[0], min(tri.Y[1], tri.Y[2])));
                            narrow = ext < NARROW_EXT;
                            wide = !narrow;
                            if (A < 0) {
                                swap12(tri);
#pragma unroll
                                for (int ch = 0; ch < 3; ++ch) { const float f = oc[1][ch]; oc[1][ch] = oc[2][ch]; oc[2][ch] = f; }
                            }
                        }
                    }
                }
            }
            if (__ballot_sync(FULL, narrow || wide) == 0u) continue;
            if (STATS) n_tri += (narrow || wide) ? 1u : 0u;
            {
                uint32_t E0[3] = {0u, 0u, 0u}, D[3] = {0u, 0u, 0u}, bbw = 0u;
                bool swapped;
                if (narrow) narrow_setup(tri.X, tri.Y, tri.q, i0, i1, j0, j1, E0, D, bbw, swapped);   // already normalised: no swap
                emit_narrow<true>(PP, env, lane, narrow, E0, D, bbw, j0, j1, tri.id2, tri.q, nullptr, oc, overflow);
            }
            emit_wide(PP, env, lane, wide, tri, j0, j1, oc, overflow);
        }
    }
    __syncwarp();
}

}  // namespace gx

namespace gx {

// ------------------------------------------------------------------------------------------------
// K1: the cull kernel.  One CTA per environment: every cluster AABB of the environment is tested against the
// frustum and the batches of the survivors are appended to the chunk-wide work list (warp-aggregated atomics).
//   PHASE 1  writes the environment table (model-view matrices N1/N2, id bases), and, when the occluder
//            phase is on (occl_pct < 100), keeps only the nearest occl_pct % of the visible clusters: a
//            256-bin histogram of the boxes' wmin gives the threshold thr[env]; clusters with wmin < thr go.
//   PHASE 2  takes the other visible clusters and drops those that the hi-Z tiles left by the first raster
//            phase prove hidden (box_occluded).
// ------------------------------------------------------------------------------------------------
template <int WARPS, int PHASE, bool STATS>
__global__ void __launch_bounds__(WARPS * 32) cull_kernel(const PipeParams PP) {
    extern __shared__ __align__(16) unsigned char smem[];
    const GxParams &P = PP.g;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NT = WARPS * 32;
    const int K = P.K;
    const int env = blockIdx.x;

    unsigned char *p = smem;
    EnvSmem es;
    es.MV = reinterpret_cast<float *>(p);          p += (size_t)(K + 1) * 48;
    es.id_base = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 2) * 4;
    es.cl_base = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 2) * 4;
    es.slot_cl = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 1) * 4;
    es.slot_mesh = reinterpret_cast<int32_t *>(p); p += (size_t)(K + 1) * 4;
    es.slot_nt = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 1) * 4;
    es.slot_nc = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 1) * 4;
    es.work = nullptr;
    __shared__ unsigned s_hist[256];
    __shared__ float s_hz[HZ_STRIDE];
    __shared__ float s_thr;

    if (PHASE == 2 && PP.env_flag[env]) return;   // overflowed in the occluder phase: single-kernel pass
    env_setup(P, env, es, tid);
    if (PHASE == 1) {
        float *g_mv = PP.env_mv + (size_t)env * (size_t)(K + 1) * 12;
        uint32_t *g_idb = PP.env_idb + (size_t)env * (size_t)(K + 1);
        for (int k = tid; k < (K + 1) * 12; k += NT) g_mv[k] = es.MV[k];
        for (int k = tid; k <= K; k += NT) g_idb[k] = es.id_base[k];
    }
    const uint32_t n_cl = es.cl_base[K + 1];
    const bool need_thr = P.cull && PP.nphase >= 3;   // the depth threshold only splits the big sub-clusters of a 3-pass scheme

    auto slot_of = [&](uint32_t g) {
        int lo = 0, hi = K;
        while (lo < hi) {   // largest slot whose first cluster index is <= g
            const int mid = (lo + hi + 1) >> 1;
            if (es.cl_base[mid] <= g) lo = mid; else hi = mid - 1;
        }
        return (uint32_t)lo;
    };

    float thr = 3.0e38f;
    if (PHASE == 1 && need_thr) {
        for (int k = tid; k < 256; k += NT) s_hist[k] = 0;
        __syncthreads();
        const float inv_bin = 256.0f / P.zfar;
        for (uint32_t g = tid; g < n_cl; g += NT) {
            const uint32_t s = slot_of(g);
            const CamBox b = cluster_box(P.clusters[es.slot_cl[s] + (g - es.cl_base[s])], es.MV + s * 12);
            if (box_in_frustum(b, P.fx, P.fy, P.znear, P.zfar))
                atomicAdd(&s_hist[(int)fminf(fmaxf(b.wmin * inv_bin, 0.0f), 255.0f)], 1u);
        }
        __syncthreads();
        if (warp == 0) {   // smallest bin edge below which at least occl_pct % of the visible clusters lie
            unsigned v[8], sum = 0;
#pragma unroll
            for (int k = 0; k < 8; ++k) { v[k] = s_hist[lane * 8 + k]; sum += v[k]; }
            unsigned inc = sum;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned a = __shfl_up_sync(0xFFFFFFFFu, inc, d);
                if (lane >= d) inc += a;
            }
            const unsigned total = __shfl_sync(0xFFFFFFFFu, inc, 31);
            const unsigned want = (total * (unsigned)PP.occl_pct + 99u) / 100u;
            unsigned run = inc - sum;
            int bin = 256;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                run += v[k];
                if (bin == 256 && run >= want) bin = lane * 8 + k;
            }
#pragma unroll
            for (int d = 16; d; d >>= 1) bin = min(bin, __shfl_xor_sync(0xFFFFFFFFu, bin, d));
            if (lane == 0) {
                s_thr = (float)(bin + 1) * (P.zfar / 256.0f);
                PP.thr[env] = s_thr;
            }
        }
        __syncthreads();
        thr = s_thr;
    }
    if (PHASE == 2) {
        thr = PP.thr[env];
        for (int k = tid; k < HZ_STRIDE; k += NT) s_hz[k] = PP.hiz[(size_t)env * HZ_STRIDE + k];
        __syncthreads();
    }

    unsigned st_tested = 0, st_drawn = 0;
    constexpr int CCH = 256;                                   // clusters per round
    constexpr int VB_CAP = CCH * GX_MAX_BATCH_PER_CLUSTER;     // batches of the visible clusters of a round
    __shared__ uint32_t s_vb[VB_CAP], s_vm[VB_CAP], s_vlo[VB_CAP], s_vhi[VB_CAP];
    __shared__ unsigned s_nvb;
    for (uint32_t c0 = 0; c0 < n_cl; c0 += CCH) {
        if (tid == 0) s_nvb = 0;
        __syncthreads();
        // step 1, one thread per cluster: frustum (and, in a later pass of the occluder scheme, hi-Z) test of the
        // cluster AABB; the batches of the survivors are listed in shared memory
        for (uint32_t g = c0 + tid; g < min(c0 + (uint32_t)CCH, n_cl); g += NT) {
            const uint32_t s = slot_of(g);
            const GxClusterDev c = P.clusters[es.slot_cl[s] + (g - es.cl_base[s])];
            bool vis = true;
            if (P.cull) {
                const CamBox b = cluster_box(c, es.MV + s * 12);
                vis = box_in_frustum(b, P.fx, P.fy, P.znear, P.zfar);
                if (PHASE == 1) {
                    if (STATS) { ++st_tested; st_drawn += vis ? 1u : 0u; }
                } else {
                    const bool occ = vis && box_occluded(b, s_hz, P.fx, P.fy, P.W, P.H, P.znear);
                    if (STATS) st_tested += occ ? 1u : 0u;   // (PHASE 2: st_tested counts the clusters proved hidden)
                    vis = vis && !occ;
                }
            } else if (STATS) { ++st_tested; ++st_drawn; }
            if (vis) {
                const uint32_t nb = min(c.nbatch, (uint32_t)GX_MAX_BATCH_PER_CLUSTER);
                const uint32_t at = atomicAdd(&s_nvb, nb);
                for (uint32_t k = 0; k < nb; ++k) {
                    s_vb[at + k] = (s << 24) | (c.batch_off + k);
                    s_vm[at + k] = 0u; s_vlo[at + k] = 0xFFFFu; s_vhi[at + k] = 0u;
                }
            }
        }
        __syncthreads();
        const unsigned nvb = s_nvb;
        // step 2 (K1b, sub-cluster culling), one thread per run of 32 triangles of a listed batch: its AABB is
        // tested against the frustum and, in the occluder scheme, classified (pass 1: big-triangle sub-clusters,
        // the cheap occluders; later passes: the rest) and tested against the hi-Z tiles
        for (unsigned idx = tid; idx < nvb * GX_SUBS_PER_BATCH; idx += NT) {
            const unsigned v = idx / GX_SUBS_PER_BATCH, r = idx % GX_SUBS_PER_BATCH;
            const uint32_t batch = s_vb[v] & 0xFFFFFFu, s = s_vb[v] >> 24;
            if ((int)r * 32 >= (int)(P.batches[batch].nv_nt >> 16)) continue;
            const GxClusterDev sb = P.subs[(size_t)batch * GX_SUBS_PER_BATCH + r];
            bool sv = true;
            if (PP.subcull || PP.phase) {
                const CamBox bx = cluster_box(sb, es.MV + s * 12);
                sv = !PP.subcull || box_in_frustum(bx, P.fx, P.fy, P.znear, P.zfar);
                if (sv && PP.phase) {
                    const int cls = sub_class(bx, P.fx, P.fy, P.W, P.H, P.znear, PP.occl_area, thr, PP.nphase);
                    sv = cls == PP.phase - 1 && (PHASE == 1 || !box_occluded(bx, s_hz, P.fx, P.fy, P.W, P.H, P.znear));
                }
            }
            if (sv) {
                atomicOr(&s_vm[v], 1u << r);
                atomicMin(&s_vlo[v], sb.batch_off);   // (fields reused: first and last vertex the run references)
                atomicMax(&s_vhi[v], sb.nbatch);
            }
        }
        __syncthreads();
        // step 3: one work item per batch that has a run left: (slot | batch, environment, mask of runs, vertex range)
        for (unsigned v0 = warp * 32; v0 < nvb; v0 += NT) {
            const unsigned v = v0 + lane;
            const bool has = v < nvb && s_vm[v] != 0u;
            const unsigned m = __ballot_sync(0xFFFFFFFFu, has);
            uint32_t base = 0;
            if (lane == 0 && m) base = atomicAdd(&PP.counters[2], (unsigned)__popc(m));
            base = __shfl_sync(0xFFFFFFFFu, base, 0);
            if (has) PP.items[base + __popc(m & ((1u << lane) - 1u))] = make_uint4(s_vb[v], (uint32_t)env, s_vm[v], s_vlo[v] | (s_vhi[v] << 16));
        }
        __syncthreads();
    }
    if (STATS) {
#pragma unroll
        for (int d = 16; d; d >>= 1) {
            st_tested += __shfl_xor_sync(0xFFFFFFFFu, st_tested, d);
            st_drawn += __shfl_xor_sync(0xFFFFFFFFu, st_drawn, d);
        }
        if (lane == 0) {
            if (PHASE == 1) {
                atomicAdd(&P.stats[GX_STAT_CLUSTERS_TESTED], (unsigned long long)st_tested);
                atomicAdd(&P.stats[GX_STAT_CLUSTERS_DRAWN], (unsigned long long)st_drawn);
            } else {
                atomicAdd(&P.stats[GX_STAT_CLUSTERS_OCCLUDED], (unsigned long long)st_tested);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// K2: the geometry kernel.  Persistent warps draw (environment, slot, batch) items from the work list; there
// is no CTA-level synchronisation at all.
// ------------------------------------------------------------------------------------------------
template <int WARPS, bool STATS>
__global__ void __launch_bounds__(WARPS * 32, GEOM_MINB) geom_kernel(const PipeParams PP) {
    extern __shared__ __align__(16) unsigned char smem[];
    const GxParams &P = PP.g;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int K = P.K;

    GeomWarpSmem ws;
    {
        unsigned char *w = smem + (size_t)warp * GEOM_WARP_SMEM;
        ws.vXY = reinterpret_cast<int2 *>(w);
        ws.vQ = reinterpret_cast<float *>(w + GX_VCAP * 8);
        ws.vC = reinterpret_cast<uint32_t *>(w + GX_VCAP * 12);
        ws.lst = w + GX_VCAP * 16;
    }
    Proj pj;
    pj.fx = P.fx; pj.fy = P.fy;
    pj.hw = 128.0f * (float)P.W; pj.hh = 128.0f * (float)P.H;

    unsigned st_in = 0, st_tri = 0;
    const unsigned n_items = PP.counters[2];
    unsigned next = 0;
    if (lane == 0) next = atomicAdd(&PP.counters[0], 1u);
    next = __shfl_sync(0xFFFFFFFFu, next, 0);
    while (next < n_items) {
        const uint4 item = PP.items[next];
        if (lane == 0) next = atomicAdd(&PP.counters[0], 1u);   // draw the following item while this one is processed
        const int env = (int)item.y;
        const uint32_t s = item.x >> 24;
        bool overflow = false;
        geom_batch<STATS>(PP, pj, item.x & 0xFFFFFFu, PP.env_mv + ((size_t)env * (size_t)(K + 1) + s) * 12,
                          PP.env_idb[(size_t)env * (size_t)(K + 1) + s], ws, env, lane, item.z, (int)(item.w & 0xFFFFu),
                          (int)(item.w >> 16), overflow, st_in, st_tri);
        if (overflow && lane == 0 && atomicExch(&PP.env_flag[env], 1u) == 0u)
            atomicAdd(&P.stats[GX_STAT_OVERFLOW_ENVS], 1ull);
        next = __shfl_sync(0xFFFFFFFFu, next, 0);
    }
    if (STATS) {
#pragma unroll
        for (int d = 16; d; d >>= 1) st_tri += __shfl_xor_sync(0xFFFFFFFFu, st_tri, d);
        if (lane == 0) {
            atomicAdd(&P.stats[GX_STAT_TRIS_IN], (unsigned long long)st_in);
            atomicAdd(&P.stats[GX_STAT_TRIS_RASTER], (unsigned long long)st_tri);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// raster order: environments sorted by record count, heaviest first (one CTA, counting sort in 256 bins), so
// that the persistent raster CTAs finish together.
// ------------------------------------------------------------------------------------------------
constexpr unsigned WIDE_COST = 1024;   // raster cost of a wide record in units of a narrow record: a whole warp walks
                                       // its (often frame-sized) bounding box block by block
__global__ void __launch_bounds__(1024) order_kernel(const PipeParams PP, const int since_phase1) {
    __shared__ unsigned hist[256];
    const int tid = threadIdx.x, N = PP.g.N * PP.bands;   // tasks: (environment, band)
    auto cost = [&](int e) {
        unsigned n = PP.cnt[2 * e], w = PP.cnt[2 * e + 1];
        if (since_phase1) { n -= PP.cnt1[2 * e]; w -= PP.cnt1[2 * e + 1]; }
        return n + WIDE_COST / 2u * w;   // (w counts two slots per wide record)
    };
    if (tid < 256) hist[tid] = 0;
    __syncthreads();
    unsigned mx_n = 0, mx_w = 0;
    for (int e = tid; e < N; e += 1024) {
        atomicAdd(&hist[255u - min(255u, cost(e) >> 7)], 1u);
        mx_n = max(mx_n, PP.cnt[2 * e]);
        mx_w = max(mx_w, PP.cnt[2 * e + 1]);
    }
    mx_n = __reduce_max_sync(0xFFFFFFFFu, mx_n);
    mx_w = __reduce_max_sync(0xFFFFFFFFu, mx_w);
    if ((tid & 31) == 0) { atomicMax(&PP.maxrec[0], mx_n); atomicMax(&PP.maxrec[1], mx_w); }
    __syncthreads();
    if (tid < 32) {   // exclusive scan of the 256 bins by one warp, 8 bins per lane
        unsigned v[8], sum = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) { v[k] = hist[tid * 8 + k]; sum += v[k]; }
        unsigned inc = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned a = __shfl_up_sync(0xFFFFFFFFu, inc, d);
            if (tid >= d) inc += a;
        }
        unsigned run = inc - sum;
#pragma unroll
        for (int k = 0; k < 8; ++k) { hist[tid * 8 + k] = run; run += v[k]; }
    }
    __syncthreads();
    for (int e = tid; e < N; e += 1024) {
        PP.order[atomicAdd(&hist[255u - min(255u, cost(e) >> 7)], 1u)] = (uint32_t)e;
    }
}

// ------------------------------------------------------------------------------------------------
// raster side
// ------------------------------------------------------------------------------------------------
struct RastWarpSmem {
    uint32_t *rec;   // [REC_WORDS * 32] SoA records of the current group (layout of gx_kernels.cuh R_*)
    uint32_t *fq;    // [FQ_CAP] covered fragments: r | (x - i0) << 5 | (y - j0) << 12
};
constexpr int RAST_WARP_SMEM = REC_WORDS * 32 * 4 + FQ_CAP * 4;
constexpr int WIDE_ROWS = 16;   // a wide record is drawn strip by strip: one draw = one strip of this many rows, by one warp

__host__ __device__ inline size_t raster_smem_bytes(int W, int H, int warps) {
    return (size_t)W * H * 8 + (size_t)warps * RAST_WARP_SMEM;
}

// N9 with the frame key (depth bits << 32 | slot index): smaller depth wins; at exactly equal depth the
// smaller (id << 1 | sub) wins, read from the stored slot's record (rare).  The final frame holds, per pixel,
// the slot of the lexicographically smallest (depth, id, sub) whatever the order of arrival.
__device__ __forceinline__ void key_min_rec(unsigned long long *slot, uint32_t dbits, uint32_t idx, uint32_t id2,
                                            const uint4 *env_recs) {
    const unsigned long long key = ((unsigned long long)dbits << 32) | idx;
    unsigned long long cur = *reinterpret_cast<volatile unsigned long long *>(slot);
    for (;;) {
        const uint32_t cd = (uint32_t)(cur >> 32);
        if (dbits > cd) return;
        if (dbits == cd) {
            const uint32_t cid2 = __ldg(reinterpret_cast<const uint32_t *>(env_recs + (size_t)(uint32_t)cur * 4) + P_ID);
            if (id2 >= cid2) return;
        }
        const unsigned long long old = atomicCAS(slot, cur, key);
        if (old == cur) return;
        cur = old;
    }
}

// load the group's records (one per lane) into the warp's SoA staging
__device__ __forceinline__ void load_group(const RastWarpSmem &ws, const uint4 *env_recs, uint32_t first, int nrec, int lane) {
    if (lane < nrec) {
        const uint4 *rp = env_recs + (size_t)(first + (uint32_t)lane) * 4;
        const uint4 u0 = __ldg(rp), u1 = __ldg(rp + 1), u2 = __ldg(rp + 2);
        ws.rec[(R_E0 + 0) * 32 + lane] = u0.x;
        ws.rec[(R_E0 + 1) * 32 + lane] = u0.y;
        ws.rec[(R_E0 + 2) * 32 + lane] = u0.z;
        ws.rec[(R_D0 + 0) * 32 + lane] = u0.w;
        ws.rec[(R_D0 + 1) * 32 + lane] = u1.x;
        ws.rec[(R_D0 + 2) * 32 + lane] = u1.y;
        ws.rec[R_BB * 32 + lane] = u1.z;
        ws.rec[R_ID * 32 + lane] = u1.w;
        ws.rec[(R_Q0 + 0) * 32 + lane] = u2.x;
        ws.rec[(R_Q0 + 1) * 32 + lane] = u2.y;
        ws.rec[(R_Q0 + 2) * 32 + lane] = u2.z;
        ws.rec[R_FA * 32 + lane] = __float_as_uint((float)(int)(u0.x + u0.y + u0.z));   // E_0 + E_1 + E_2 = A
    }
    __syncwarp();
}

// K4b: depth (N7) and resolve (N9) for the queued fragments, one per lane
__device__ __forceinline__ void shade_queue_p(const RastWarpSmem &ws, int qn, int W, float zfar, unsigned long long *fb,
                                              uint32_t first, const uint4 *env_recs, int lane) {
    for (int f = lane; f < qn; f += 32) {
        const uint32_t en = ws.fq[f];
        const int r = (int)(en & 31u), a = (int)((en >> 5) & 127u), b = (int)((en >> 12) & 127u);
        const uint32_t bb = ws.rec[R_BB * 32 + r];
        const int x = (int)(bb & 127u) + a, y = (int)((bb >> 7) & 127u) + b;
        unsigned long long *slot = &fb[fb_index(x, y, W)];
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
        key_min_rec(slot, __float_as_uint(depth), first + (uint32_t)r, ws.rec[R_ID * 32 + r], env_recs);
    }
    __syncwarp();
}

// K3: the bounding boxes of the group's records are cut into slots of 4 pixels of one row.  group_slots returns
// the lane's exclusive prefix of slot counts (Pex, record = lane) and the group's total T.
// With hz != NULL (second raster phase) a record whose nearest vertex is strictly behind the hi-Z value of
// every 8x8 tile its bounding box touches gets no slots: none of its fragments could win N9.
template <int SW>
__device__ __forceinline__ int group_slots(const RastWarpSmem &ws, int nrec, int lane, const float *hz, int &Pex,
                                           unsigned &skip, unsigned &n_culled) {
    const unsigned FULL = 0xFFFFFFFFu;
    int ns = 0;
    bool culled = false;
    if (lane < nrec) {
        const uint32_t bb = ws.rec[R_BB * 32 + lane];
        const int w = (int)((bb >> 14) & 127u) + 1, h = (int)((bb >> 21) & 127u) + 1;
        ns = h * ((w + SW - 1) / SW);
        if (hz) {
            const int i0 = (int)(bb & 127u), j0 = (int)((bb >> 7) & 127u);
            const int tx0 = i0 >> 3, tx1 = (i0 + w - 1) >> 3, ty0 = j0 >> 3, ty1 = (j0 + h - 1) >> 3;
            if ((tx1 - tx0 + 1) * (ty1 - ty0 + 1) <= 6) {
                float zmax = 0.0f;
                for (int ty = ty0; ty <= ty1; ++ty)
                    for (int tx = tx0; tx <= tx1; ++tx) zmax = fmaxf(zmax, hz[ty * 16 + tx]);
                const float qmax = fmaxf(__uint_as_float(ws.rec[(R_Q0 + 0) * 32 + lane]),
                                         fmaxf(__uint_as_float(ws.rec[(R_Q0 + 1) * 32 + lane]),
                                               __uint_as_float(ws.rec[(R_Q0 + 2) * 32 + lane])));
                // every depth of the triangle is >= 1/qmax (N7, up to a few ulp): hidden iff 1/qmax > zmax with margin
                if (qmax * zmax < 1.0f - 1e-5f) { ns = 0; culled = true; ++n_culled; }
            }
        }
    }
    skip = __ballot_sync(FULL, culled);   // records without slots: the slot walk steps over them
    int inc = ns;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(FULL, inc, d);
        if (lane >= d) inc += v;
    }
    Pex = inc - ns;
    return __shfl_sync(FULL, inc, 31);
}

// K3 + K4a: coverage of the slots [S0, S1) of the warp's group.  The slots are dealt to the lanes in equal
// contiguous runs (a lane walks through its run, moving to the next record when one is exhausted), so that
// lanes stay busy whatever the mix of triangle sizes.  The covered pixels of one pass are appended to the
// fragment queue with four ballots and shaded densely by shade_queue_p.
template <bool STATS, int SW>
__device__ __forceinline__ void raster_slots(const RastWarpSmem &ws, int Pex, unsigned skip, int S0, int S1, int W, float zfar,
                                             unsigned long long *fb, uint32_t first, const uint4 *env_recs, int lane,
                                             unsigned &n_frag) {
    const unsigned FULL = 0xFFFFFFFFu;
    const unsigned lt = (1u << lane) - 1u;
    const int per = (S1 - S0 + 31) >> 5;
    const int s0 = S0 + lane * per;
    const int n = max(0, min(per, S1 - s0));
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
            E0[e] = (int)ws.rec[(R_E0 + e) * 32 + rr] - (int)((bb >> (28 + e)) & 1u);
            const uint32_t d = ws.rec[(R_D0 + e) * 32 + rr];
            dx[e] = (int)d >> 16;
            dy[e] = (int)(short)(d & 0xFFFFu);
        }
        w = (int)((bb >> 14) & 127u) + 1;
        h = (int)((bb >> 21) & 127u) + 1;
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
            m4 &= (1u << min(SW, w - a)) - 1u;   // pixels beyond the bounding box
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
                shade_queue_p(ws, qn, W, zfar, fb, first, env_recs, lane);
                qn = 0;
            }
            uint32_t en = (uint32_t)r | ((uint32_t)a << 5) | ((uint32_t)row << 12);
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
        shade_queue_p(ws, qn, W, zfar, fb, first, env_recs, lane);
    }
}

// wide records: one triangle at a time, the whole warp walks its bounding box in 8x4-pixel blocks with the
// int64 edge functions of N6
template <bool STATS>
__device__ __forceinline__ void raster_wide(const uint4 *env_recs, uint32_t slot0, int ntri, int W, int H, int y_lo, int bh,
                                            int y_fb, float zfar, unsigned long long *fb, int lane, unsigned &n_frag) {
    const unsigned FULL = 0xFFFFFFFFu;
    Tri tri;
#pragma unroll
    for (int k = 0; k < 3; ++k) { tri.X[k] = 0; tri.Y[k] = 0; tri.q[k] = 0.0f; }
    tri.id2 = 0;
    if (lane < ntri) {
        const uint4 *rp = env_recs + (size_t)(slot0 + 2u * (uint32_t)lane) * 4;
        const uint4 u0 = __ldg(rp), u1 = __ldg(rp + 1), u2 = __ldg(rp + 2);
        tri.X[0] = (int)u0.x; tri.X[1] = (int)u0.y; tri.X[2] = (int)u0.z;
        tri.Y[0] = (int)u0.w; tri.Y[1] = (int)u1.x; tri.Y[2] = (int)u1.y;
        tri.id2 = u1.w;
        tri.q[0] = __uint_as_float(u2.x); tri.q[1] = __uint_as_float(u2.y); tri.q[2] = __uint_as_float(u2.z);
    }
    for (int src = 0; src < ntri; ++src) {
        Tri bt;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            bt.X[k] = __shfl_sync(FULL, tri.X[k], src);
            bt.Y[k] = __shfl_sync(FULL, tri.Y[k], src);
            bt.q[k] = __shfl_sync(FULL, tri.q[k], src);
        }
        bt.id2 = __shfl_sync(FULL, tri.id2, src);
        int bi0, bi1, bj0, bj1;
        pixel_bbox(bt.X, bt.Y, W, H, bi0, bi1, bj0, bj1);
        bj0 = max(bj0, y_lo);                 // the strip's rows only (frame rows y_lo .. y_lo + bh - 1; the band starts at y_fb)
        bj1 = min(bj1, y_lo + bh - 1);
        Edges BE;
        edge_setup(bt, area2(bt), BE);   // orientation-normalised by the geometry kernel: area > 0
        const int lx = lane & 7, ly = lane >> 3;
        const uint32_t idx = slot0 + 2u * (uint32_t)src;
        for (int by = bj0 >> 2; by <= (bj1 >> 2); ++by)
            for (int bx = bi0 >> 3; bx <= (bi1 >> 3); ++bx) {
                const int i = bx * 8 + lx, j = by * 4 + ly;
                float f[3], num, depth;
                if (!cover_depth(BE, bt.q, i, j, f, num, depth)) continue;
                if (STATS) ++n_frag;
                if (depth > zfar) continue;
                key_min_rec(&fb[fb_index(i, j - y_fb, W)], __float_as_uint(depth), idx, bt.id2, env_recs);
            }
    }
    __syncwarp();
}

// K5a: colour (N8) and id of the winning record at pixel (x, y) of the band whose first frame row is y_lo
__device__ __forceinline__ uint32_t resolve_rec(const uint4 *env_recs, uint32_t cap_n, uint32_t idx, int x, int y, int y_lo,
                                                bool want_rgb, uint32_t &id) {
    const uint4 *rp = env_recs + (size_t)idx * 4;
    const uint4 u1 = __ldg(rp + 1);
    id = u1.w >> 1;
    if (!want_rgb) return 0u;
    const uint4 u0 = __ldg(rp), u2 = __ldg(rp + 2);
    const float q[3] = {__uint_as_float(u2.x), __uint_as_float(u2.y), __uint_as_float(u2.z)};
    float f[3], c[3][3];
    bool fcol = true;
    if (idx < cap_n) {
        const uint32_t bb = u1.z;
        const int a = x - (int)(bb & 127u), b = y - (int)((bb >> 7) & 127u);
        const uint32_t D[3] = {u0.w, u1.x, u1.y};
        const uint32_t E[3] = {u0.x, u0.y, u0.z};
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const int dx = (int)D[e] >> 16, dy = (int)(short)(D[e] & 0xFFFFu);
            f[e] = (float)((int)E[e] + ((b * dx - a * dy) << 8));
        }
        fcol = (bb & BB_FLOATCOL) != 0u;
        if (!fcol) {
            const uint4 u3 = __ldg(rp + 3);
            const uint32_t col[3] = {u2.w, u3.x, u3.y};
#pragma unroll
            for (int v = 0; v < 3; ++v)
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) c[v][ch] = (float)((col[v] >> (8 * ch)) & 0xFFu);
        }
    } else {
        Tri t;
        t.X[0] = (int)u0.x; t.X[1] = (int)u0.y; t.X[2] = (int)u0.z;
        t.Y[0] = (int)u0.w; t.Y[1] = (int)u1.x; t.Y[2] = (int)u1.y;
        t.q[0] = q[0]; t.q[1] = q[1]; t.q[2] = q[2];
        Edges E;
        edge_setup(t, area2(t), E);
        float num, depth;
        cover_depth(E, t.q, x, y + y_lo, f, num, depth);   // covered by construction: this triangle won the pixel
    }
    if (fcol) {
        const uint4 v1 = __ldg(rp + 5), v2 = __ldg(rp + 6), v3 = __ldg(rp + 7);
        c[0][0] = __uint_as_float(v1.w); c[0][1] = __uint_as_float(v2.x); c[0][2] = __uint_as_float(v2.y);
        c[1][0] = __uint_as_float(v2.z); c[1][1] = __uint_as_float(v2.w); c[1][2] = __uint_as_float(v3.x);
        c[2][0] = __uint_as_float(v3.y); c[2][1] = __uint_as_float(v3.z); c[2][2] = __uint_as_float(v3.w);
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


// ------------------------------------------------------------------------------------------------
// the raster kernel.  PHASE 0: draw all records of the task and write the images.  PHASE 1 (first occluder
// pass): draw the records present so far, then leave the frame keys, the hi-Z tiles and the record counts in
// global memory.  PHASE 2 (last pass): start from those keys, draw only the records appended since, skipping
// records the hi-Z tiles prove hidden, and write the images.  PHASE 3 (middle pass): start like 2, end like 1.
// ------------------------------------------------------------------------------------------------
template <int WARPS, int MINB, int PHASE, bool STATS>
__global__ void __launch_bounds__(WARPS * 32, MINB) raster_kernel(const PipeParams PP) {
    extern __shared__ __align__(16) unsigned char smem[];
    const GxParams &P = PP.g;
    constexpr int SW = (PHASE == 2 || PHASE == 3) ? 4 : 8;            // pixels per slot: the occluder pass draws big triangles
    constexpr bool LOAD = PHASE == 2 || PHASE == 3;   // start from the previous pass's frame keys and hi-Z tiles
    constexpr bool DUMP = PHASE == 1 || PHASE == 3;   // leave frame keys, hi-Z tiles and record counts for the next pass
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NT = WARPS * 32;
    const int W = P.W, H = P.H, npix = W * H;
    const int bh = PP.bh, npb = W * bh;   // rows and pixels of one band: the CTA's frame

    unsigned long long *fb = reinterpret_cast<unsigned long long *>(smem);
    RastWarpSmem ws;
    ws.rec = reinterpret_cast<uint32_t *>(smem + (size_t)npb * 8 + (size_t)warp * RAST_WARP_SMEM);
    ws.fq = ws.rec + REC_WORDS * 32;

    __shared__ int s_env;
    __shared__ unsigned s_next, s_next_b, s_big, s_classified;
    constexpr int BIG_CAP = 16 * WARPS;     // entries of the pass-B list
    __shared__ uint2 s_big_list[BIG_CAP];   // (group, first chunk) of the groups left to pass B
    __shared__ float s_hz[HZ_STRIDE];
    __shared__ unsigned long long s_frag, s_culled;

    unsigned st_frag = 0, st_culled = 0;
    if (STATS && tid == 0) { s_frag = 0; s_culled = 0; }
    const uint4 ones = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
    if (!LOAD) {
        uint4 *f4 = reinterpret_cast<uint4 *>(fb);
        for (int k = tid; k < npb / 2; k += NT) f4[k] = ones;
    }
    const bool want_rgb = P.rgb != nullptr || P.obs != nullptr;
    const uint32_t cap_n = (uint32_t)PP.cap_n;

    for (;;) {
        if (tid == 0) {   // next task: (environment, band), heaviest first
            const unsigned k = atomicAdd(&PP.counters[1], 1u);
            s_env = k < (unsigned)(P.N * PP.bands) ? (int)PP.order[k] : -1;
            s_next = 0; s_next_b = 0; s_big = 0; s_classified = 0;
        }
        __syncthreads();
        const int v = s_env;
        if (v < 0) break;
        const int env = v / PP.bands, y_lo = (v - env * PP.bands) * bh;
        const float *hz = LOAD ? s_hz + (y_lo >> 3) * 16 : nullptr;
        if (PP.env_flag[env]) {   // overflowed its pool segment: left to the single-kernel pass
            __syncthreads();
            continue;
        }
        const uint4 *env_recs = PP.recs + (size_t)v * (size_t)(PP.cap_n + PP.cap_w) * 4;
        const uint32_t n_n = PP.cnt[2 * v], n_w = PP.cnt[2 * v + 1] >> 1;
        const uint32_t b_n = LOAD ? PP.cnt1[2 * v] : 0u, b_w = LOAD ? PP.cnt1[2 * v + 1] >> 1 : 0u;
        const uint32_t wu = (uint32_t)(bh + WIDE_ROWS - 1) / WIDE_ROWS;   // strips of WIDE_ROWS rows per band
        const uint32_t g_n = (n_n - b_n + 31u) >> 5, g_w = (n_w - b_w) * wu;   // one draw = one strip of one wide record
        if (LOAD) {   // the previous pass's frame and hi-Z tiles
            const uint4 *src = reinterpret_cast<const uint4 *>(PP.frames + (size_t)v * npb);
            uint4 *f4 = reinterpret_cast<uint4 *>(fb);
            for (int k = tid; k < npb / 2; k += NT) f4[k] = __ldg(src + k);
            for (int k = tid; k < HZ_STRIDE; k += NT) s_hz[k] = PP.hiz[(size_t)env * HZ_STRIDE + k];
            __syncthreads();
        }

        // ---- K3 + K4, pass A: groups of 32 records, drawn dynamically by the warps.  A group of more than
        // big_slots slots is only registered: (list index, first chunk) come from one packed atomic, so the
        // list is ordered by first chunk.  Every group counts itself as classified as soon as that is decided.
        for (;;) {
            unsigned g = 0;
            if (lane == 0) g = atomicAdd(&s_next, 1u);
            g = __shfl_sync(0xFFFFFFFFu, g, 0);
            if (g >= g_n + g_w) break;
            if (g >= g_w) {
                const uint32_t pos = (g - g_w) * 32u;
                const int nrec = (int)min(32u, n_n - b_n - pos);
                const uint32_t first = b_n + pos;
                load_group(ws, env_recs, first, nrec, lane);
                int Pex;
                unsigned skip;
                const int T = group_slots<SW>(ws, nrec, lane, hz, Pex, skip, st_culled);
                const bool big = T > PP.big_slots;
                unsigned full = 0;
                if (lane == 0) {
                    if (big) {
                        const unsigned nch = (unsigned)(T + PP.chunk_slots - 1) / (unsigned)PP.chunk_slots;
                        const unsigned old = atomicAdd(&s_big, (1u << 20) | nch);
                        if ((old >> 20) < (unsigned)BIG_CAP) s_big_list[old >> 20] = make_uint2(g - g_w, old & 0xFFFFFu);
                        else full = 1;
                    }
                    __threadfence_block();
                    atomicAdd(&s_classified, 1u);   // this group's entry (if any) is in the list
                }
                // small group, or list full: drawn here, whole
                if ((!big || __shfl_sync(0xFFFFFFFFu, full, 0)) && T)
                    raster_slots<STATS, SW>(ws, Pex, skip, 0, T, W, P.zfar, fb, first, env_recs, lane, st_frag);
            } else {   // wide records first: they reach the near plane and hide the most
                if (lane == 0) atomicAdd(&s_classified, 1u);
                const uint32_t t0 = b_w + g / wu, strip = g % wu;
                const int ys = y_lo + (int)strip * WIDE_ROWS;
                raster_wide<STATS>(env_recs, cap_n + 2u * t0, 1, W, H, ys, min(WIDE_ROWS, y_lo + bh - ys), y_lo, P.zfar, fb, lane, st_frag);
            }
        }
        // No barrier between the passes: a warp that finds no group left waits only until every group has been
        // classified (each is, right after it is loaded), not until the small ones have been drawn.
        if (lane == 0)
            while (*reinterpret_cast<volatile unsigned *>(&s_classified) < g_n + g_w) __nanosleep(32);
        __syncwarp();
        __threadfence_block();
        // ---- pass B: the big groups, in chunks of chunk_slots slots drawn dynamically -----------------
        {
            const unsigned packed = *reinterpret_cast<volatile unsigned *>(&s_big);
            const unsigned n_big = min(packed >> 20, (unsigned)BIG_CAP), n_chunks = packed & 0xFFFFFu;
            for (;;) {
                unsigned c = 0;
                if (lane == 0) c = atomicAdd(&s_next_b, 1u);
                c = __shfl_sync(0xFFFFFFFFu, c, 0);
                if (c >= n_chunks) break;
                unsigned lo = 0, hi = n_big - 1;   // last entry whose first chunk is <= c
                while (lo < hi) {
                    const unsigned mid = (lo + hi + 1) >> 1;
                    if (s_big_list[mid].y <= c) lo = mid; else hi = mid - 1;
                }
                const uint2 en = s_big_list[lo];
                const uint32_t pos = en.x * 32u;
                const int nrec = (int)min(32u, n_n - b_n - pos);
                const uint32_t first = b_n + pos;
                load_group(ws, env_recs, first, nrec, lane);
                int Pex;
                unsigned skip, dummy = 0;
                const int T = group_slots<SW>(ws, nrec, lane, hz, Pex, skip, dummy);
                const int S0 = (int)(c - en.y) * PP.chunk_slots;   // chunks of entries a full list dropped land beyond T
                if (S0 < T) raster_slots<STATS, SW>(ws, Pex, skip, S0, min(T, S0 + PP.chunk_slots), W, P.zfar, fb, first, env_recs, lane, st_frag);
            }
        }
        __syncthreads();

        if (DUMP) {
            // ---- occluder pass: hi-Z tiles (max depth per 8x8 tile, +inf where background shows), the frame
            // keys and the record counts go to global memory; the frame is reset for the next environment
            const int tw = W >> 3, th = bh >> 3, ty0 = y_lo >> 3;   // the band's tile rows are ty0 .. ty0 + th - 1
            for (int u = warp; u < th * 2; u += WARPS) {   // a warp takes half a row of tiles; a lane, 2 of a tile's 64 keys
                const int ty = u >> 1, j = ty * 8 + (lane >> 2);
                const unsigned long long *row = fb + j * W;
                const int sw = (j & 1) << 3, i0 = (lane & 3) * 2;
                const int tx_lo = (u & 1) ? (tw >> 1) : 0, tx_hi = (u & 1) ? tw : (tw >> 1);
                for (int tx = tx_lo; tx < tx_hi; ++tx) {
                    const uint4 v = *reinterpret_cast<const uint4 *>(row + ((tx * 8 + i0) ^ sw));   // depth bits in .y, .w
                    const unsigned d = __reduce_max_sync(0xFFFFFFFFu, max(v.y, v.w));
                    if (lane == 0) s_hz[ty * 16 + tx] = d == 0xFFFFFFFFu ? __int_as_float(0x7F800000) : __uint_as_float(d);
                }
            }
            __syncthreads();
            float *g_hz = PP.hiz + (size_t)env * HZ_STRIDE;
            for (int t = tid; t < th * 16; t += NT) g_hz[ty0 * 16 + t] = s_hz[t];
            // 32x32-pixel tiles: max over 4x4 of the above (a band of several bands is a multiple of 32 rows high)
            for (int t = tid; t < ((th + 3) >> 2) * 4; t += NT) {
                const int by = t >> 2, bx = t & 3;
                float z = 0.0f;
                for (int ty = by * 4; ty < min(by * 4 + 4, th); ++ty)
                    for (int tx = bx * 4; tx < min(bx * 4 + 4, tw); ++tx) z = fmaxf(z, s_hz[ty * 16 + tx]);
                g_hz[256 + ((ty0 >> 2) + by) * 4 + bx] = z;
            }
            uint4 *dst = reinterpret_cast<uint4 *>(PP.frames + (size_t)v * npb);
            uint4 *f4 = reinterpret_cast<uint4 *>(fb);
            for (int k = tid; k < npb / 2; k += NT) { dst[k] = f4[k]; if (!LOAD) f4[k] = ones; }
            if (tid < 2) PP.cnt1[2 * v + tid] = PP.cnt[2 * v + tid];
        } else {
            // ---- K5: resolve the winners, write RGB / depth / id as 16-byte stores, reset the frame ------
            const size_t out0 = (size_t)env * npix + (size_t)y_lo * W;   // first pixel of the band in the outputs
            for (int k = tid; k < npb / 4; k += NT) {
                const int pix = k * 4;
                const int j = pix / W, i = pix - j * W;
                const int a = fb_index(i, j, W);          // 4-aligned columns stay contiguous under the XOR
                uint4 *slot = reinterpret_cast<uint4 *>(&fb[a]);
                const uint4 v0 = slot[0], v1 = slot[1];
                if (PHASE == 0) { slot[0] = ones; slot[1] = ones; }   // (PHASE 2 reloads the frame per environment)
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
                        if (want_rgb || P.id) col[m] = resolve_rec(env_recs, cap_n, idx[m], i + m, j, y_lo, want_rgb, id[m]);
                    }
                }
                if (P.depth) *reinterpret_cast<float4 *>(P.depth + out0 + pix) = d;
                if (P.obs) store_obs4(P.obs + (size_t)env * 4 * npix, (size_t)npix, (size_t)y_lo * W + pix, col, dp, P.obs_dmin, P.obs_range);
                if (P.id) *reinterpret_cast<uint4 *>(P.id + out0 + pix) = make_uint4(id[0], id[1], id[2], id[3]);
                if (P.rgb) {
                    // 4 pixels = 12 bytes = 3 words per lane; 4 lanes hold 48 bytes = three 16-byte stores
                    const uint32_t w0 = (col[0] & 0xFFFFFFu) | (col[1] << 24);
                    const uint32_t w1 = ((col[1] >> 8) & 0xFFFFu) | (col[2] << 16);
                    const uint32_t w2 = ((col[2] >> 16) & 0xFFu) | (col[3] << 8);
                    const int g = lane & 3, gb = lane & ~3;
                    uint32_t o[4];
    #pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        const int m = 4 * g + r;          // word of the group's 12-word stream (g < 3)
                        const int src = gb + (m / 3) % 4, wsel = m % 3;
                        const uint32_t a0 = __shfl_sync(0xFFFFFFFFu, w0, src), a1 = __shfl_sync(0xFFFFFFFFu, w1, src),
                                       a2 = __shfl_sync(0xFFFFFFFFu, w2, src);
                        o[r] = wsel == 0 ? a0 : (wsel == 1 ? a1 : a2);
                    }
                    if (g < 3) {
                        uint8_t *dst = P.rgb + (out0 + (size_t)(pix - 4 * g)) * 3 + 16 * g;
                        *reinterpret_cast<uint4 *>(dst) = make_uint4(o[0], o[1], o[2], o[3]);
                    }
                }
            }
        }
        __syncthreads();
    }

    if (STATS) {
        atomicAdd(&s_frag, (unsigned long long)st_frag);
        atomicAdd(&s_culled, (unsigned long long)st_culled);
        __syncthreads();
        if (tid == 0) {
            atomicAdd(&P.stats[GX_STAT_FRAGMENTS], s_frag);
            atomicAdd(&P.stats[GX_STAT_RECORDS_OCCLUDED], s_culled);
        }
    }
}

}  // namespace gx
