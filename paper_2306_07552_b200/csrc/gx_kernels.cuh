// gx_kernels.cuh -- the render kernel of the batch RGBD rasteriser (sm_100a).
//
// One persistent CTA per SM renders one environment at a time ("A single ... renderer instance
// renders all environments").  A 128x128 frame of 64-bit (depth, id) keys is 128 KB and fits the 227 KB of
// shared memory a B200 CTA may own, so the whole frame is the raster tile: there is no triangle record
// stream through HBM and no per-tile binning pass.  Stages inside the kernel:
//   K1 cull     : per environment, every cluster AABB against the view frustum -> compact work list in smem
//   K2 geometry : one warp per batch: vertex transform + 1/256-px snap into warp-private smem, then per
//                 triangle the pixel-centre bounding-box reject; survivors are ballot-compacted
//   K3 bin      : survivors are sorted by size class: small ones are shaded by their own lane, big ones are
//                 broadcast and shaded by the whole warp in 8x4-pixel blocks
//   K4 raster   : integer edge functions + top-left rule, depth = fA/num, 64-bit CAS-min into the smem frame
//   K5 write    : resolve colour of the winning triangle per pixel, then 16-byte stores of RGB and depth
// Arithmetic follows DESIGN.md section 3 (N1-N9) operation by operation; compiled with -fmad=false so that
// only the fmaf() calls written here fuse.
#pragma once
#include <cuda_fp16.h>
#include "gx_types.h"

namespace gx {

constexpr unsigned long long KEY_BG = 0xFFFFFFFFFFFFFFFFull;
constexpr int X_OUT = (int)0x80000000;   // staged X of a vertex behind the near plane
constexpr int WORK_CAP = 1024;           // work items (batches) per cull chunk; clusters per chunk = P.cull_chunk
constexpr int SMALL_MAX_PX = 6;          // bounding boxes up to this many pixels are shaded by one lane
constexpr int KMAX = 254;

struct CamVert { float xc, yc, w; };

// N3: camera-space vertex.  M = 12 floats, row-major 3x4 model-view.
__device__ __forceinline__ CamVert xform(const float *M, float x, float y, float z) {
    CamVert v;
    v.xc = fmaf(M[2], z, fmaf(M[1], y, fmaf(M[0], x, M[3])));
    v.yc = fmaf(M[6], z, fmaf(M[5], y, fmaf(M[4], x, M[7])));
    float zc = fmaf(M[10], z, fmaf(M[9], y, fmaf(M[8], x, M[11])));
    v.w = -zc;
    return v;
}

struct Proj { float fx, fy, hw, hh; };

// N5: projection and snap to 1/256 pixel (round-half-even).  q = 1/w correctly rounded.
__device__ __forceinline__ void project(const Proj &P, float xc, float yc, float w, int &X, int &Y, float &q) {
    const float LIM = 268435456.0f;  // 2^28
    q = 1.0f / w;
    float Xf = fmaf((P.fx * xc) * q, P.hw, P.hw);
    float Yf = fmaf(-((P.fy * yc) * q), P.hh, P.hh);
    Xf = fminf(fmaxf(Xf, -LIM), LIM);
    Yf = fminf(fmaxf(Yf, -LIM), LIM);
    X = __float2int_rn(Xf);
    Y = __float2int_rn(Yf);
}

// N4: new vertex on the edge from an inside vertex to an outside vertex (always computed in that direction).
__device__ __forceinline__ float clip_t(float w_in, float w_out, float znear) { return (w_in - znear) / (w_in - w_out); }
__device__ __forceinline__ float clip_lerp(float t, float a_in, float a_out) { return fmaf(t, a_out - a_in, a_in); }

// fb layout: row-linear, with bit 3 of the column XORed with bit 0 of the row, so that an aligned 8x4 block
// of 64-bit keys touches every bank exactly twice (two wavefronts, the minimum) and a row segment stays a
// contiguous run.
__device__ __forceinline__ int fb_index(int i, int j, int W) { return j * W + (i ^ ((j & 1) << 3)); }

// N11: packed policy observation of 4 consecutive pixels of one row: planes R, G, B =
// binary16(c / 255.0f), plane D = binary16((clamp(depth, dmin, dmin + range) - dmin) / range); all float32
// operations, round-to-nearest-even conversions.  obs points at plane 0 of the environment, pix = y * W + x.
__device__ __forceinline__ void store_obs4(uint16_t *obs, size_t npix, size_t pix, const uint32_t col[4], const float d[4],
                                           float dmin, float range) {
#pragma unroll
    for (int ch = 0; ch < 4; ++ch) {
        unsigned short h[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            float v;
            if (ch < 3) v = (float)((col[m] >> (8 * ch)) & 0xFFu) / 255.0f;
            else v = (fminf(fmaxf(d[m], dmin), dmin + range) - dmin) / range;
            h[m] = __half_as_ushort(__float2half_rn(v));
        }
        *reinterpret_cast<uint2 *>(obs + (size_t)ch * npix + pix) =
            make_uint2((uint32_t)h[0] | ((uint32_t)h[1] << 16), (uint32_t)h[2] | ((uint32_t)h[3] << 16));
    }
}

// st.shared.u32 [addr], v if pred != 0 (a predicated store, no branch)
__device__ __forceinline__ void sts_if(uint32_t addr, uint32_t v, uint32_t pred) {
    asm volatile("{ .reg .pred p; setp.ne.u32 p, %2, 0; @p st.shared.u32 [%0], %1; }" ::"r"(addr), "r"(v), "r"(pred) : "memory");
}

__device__ __forceinline__ void key_min(unsigned long long *slot, unsigned long long key) {
    unsigned long long cur = *reinterpret_cast<volatile unsigned long long *>(slot);
    while (key < cur) {
        unsigned long long old = atomicCAS(slot, cur, key);
        if (old == cur) break;
        cur = old;
    }
}

// A post-clip triangle ready for N6-N9: snapped corners, q = 1/w per corner, packed id (id << 1 | sub).
struct Tri {
    int X[3], Y[3];
    float q[3];
    unsigned id2;
};

// Edge setup of N6 for an orientation-normalised triangle (A > 0).  Edge e runs from vertex (e+1)%3 to
// vertex (e+2)%3; bias_e = 0 for a top-left edge, 1 otherwise, so that "covered" is E_e >= bias_e.
struct Edges {
    int dx[3], dy[3], Xa[3], Ya[3], bias[3];
    float fA;
    bool narrow;  // A < 2^31: every E_e of a covered pixel fits int32
};

__device__ __forceinline__ long long area2(const Tri &t) {
    return (long long)(t.X[1] - t.X[0]) * (long long)(t.Y[2] - t.Y[0]) -
           (long long)(t.Y[1] - t.Y[0]) * (long long)(t.X[2] - t.X[0]);
}

__device__ __forceinline__ void swap12(Tri &t) {
    int a = t.X[1]; t.X[1] = t.X[2]; t.X[2] = a;
    a = t.Y[1]; t.Y[1] = t.Y[2]; t.Y[2] = a;
    float f = t.q[1]; t.q[1] = t.q[2]; t.q[2] = f;
}

__device__ __forceinline__ void edge_setup(const Tri &t, long long A, Edges &E) {
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        const int a = (e + 1) % 3, b = (e + 2) % 3;
        E.Xa[e] = t.X[a];
        E.Ya[e] = t.Y[a];
        E.dx[e] = t.X[b] - t.X[a];   // |X| <= 2^28, so the difference fits int32
        E.dy[e] = t.Y[b] - t.Y[a];
        const bool tl = (E.dy[e] < 0) || (E.dy[e] == 0 && E.dx[e] > 0);
        E.bias[e] = tl ? 0 : 1;
    }
    E.fA = (float)A;
    E.narrow = A < 2147483648ll;
}

// N6 coverage + N7 depth at pixel (i, j).  Returns true and the depth if the pixel centre is covered.
// f[] receives the three edge values as floats (weights of vertices 0, 1, 2).
__device__ __forceinline__ bool cover_depth(const Edges &E, const float q[3], int i, int j, float f[3], float &num,
                                            float &depth) {
    const int px = (i << 8) + 128, py = (j << 8) + 128;
    long long Ev[3];
    bool cov = true;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        Ev[e] = (long long)E.dx[e] * (long long)(py - E.Ya[e]) - (long long)E.dy[e] * (long long)(px - E.Xa[e]);
        cov = cov && (Ev[e] >= (long long)E.bias[e]);
    }
    if (!cov) return false;
    if (E.narrow) {
#pragma unroll
        for (int e = 0; e < 3; ++e) f[e] = (float)(int)Ev[e];
    } else {
#pragma unroll
        for (int e = 0; e < 3; ++e) f[e] = (float)Ev[e];
    }
    num = fmaf(f[2], q[2], fmaf(f[1], q[1], f[0] * q[0]));
    depth = E.fA / num;
    return true;
}

// Pixel-centre bounding box of N6 (exact), clamped to the image.  Returns false if it is empty.
__device__ __forceinline__ bool pixel_bbox(const int X[3], const int Y[3], int W, int H, int &i0, int &i1, int &j0,
                                           int &j1) {
    const int Xmin = min(X[0], min(X[1], X[2])), Xmax = max(X[0], max(X[1], X[2]));
    const int Ymin = min(Y[0], min(Y[1], Y[2])), Ymax = max(Y[0], max(Y[1], Y[2]));
    i0 = max((Xmin + 127) >> 8, 0);
    i1 = min((Xmax - 128) >> 8, W - 1);
    j0 = max((Ymin + 127) >> 8, 0);
    j1 = min((Ymax - 128) >> 8, H - 1);
    return i0 <= i1 && j0 <= j1;
}

}  // namespace gx

namespace gx {

// ------------------------------------------------------------------------------------------------
// per-environment context in shared memory
// ------------------------------------------------------------------------------------------------
struct EnvSmem {
    float *MV;            // [(K+1)*12] model-view per slot; slot 0 = static mesh (MV = V)
    uint32_t *id_base;    // [K+2] first triangle id of slot s; [K+1] = triangles in the environment
    uint32_t *cl_base;    // [K+2] first cluster-space index of slot s; [K+1] = clusters in the environment
    uint32_t *slot_cl;    // [K+1] global index of the slot's first cluster
    int32_t *slot_mesh;   // [K+1] global mesh index (static first), -1 = empty slot
    uint32_t *slot_nt;    // [K+1]
    uint32_t *slot_nc;    // [K+1]
    uint32_t *work;       // [WORK_CAP] slot << 24 | global batch index
};

// Record of a set-up "narrow" triangle (bounding-box extent < NARROW_EXT sub-pixel units in x and y, so every
// edge value at a pixel centre of its bounding box fits int32).  Stored SoA: word k of record r at rec[k*32+r].
enum { R_E0 = 0, R_E1, R_E2,   // E_e at the bounding-box origin pixel (i0, j0)
       R_D0, R_D1, R_D2,       // edge deltas: dx_e << 16 | (dy_e & 0xFFFF)
       R_Q0, R_Q1, R_Q2,       // q = 1/w of vertices 0, 1, 2 (after orientation normalisation)
       R_FA,                   // (float)A
       R_ID,                   // id << 1 | sub
       R_BB,                   // i0 | j0 << 7 | (w-1) << 14 | (h-1) << 21 | bias bits << 28
       REC_WORDS };
constexpr int NARROW_EXT = 30000;   // 2 * 30000 * (30000 + 3*256) < 2^31
constexpr int FQ_CAP = 256;         // fragment queue entries per warp

struct WarpSmem {
    int2 *vXY;            // [GX_VCAP] snapped position, X = X_OUT if behind the near plane
    float *vQ;            // [GX_VCAP] 1/w
    unsigned char *lst;   // [256] batch-local triangle indices: narrow survivors from the front, slow-path
                          //       triangles (wide, or straddling the near plane) from the back
    uint32_t *rec;        // [REC_WORDS * 32] records of the current group
    uint32_t *fq;         // [FQ_CAP] covered fragments: r | (x - i0) << 5 | (y - j0) << 12
};

constexpr int WARP_SMEM_BYTES = GX_VCAP * 8 + GX_VCAP * 4 + 256 + REC_WORDS * 32 * 4 + FQ_CAP * 4;

__host__ __device__ inline size_t env_smem_bytes(int K) {
    return (size_t)(K + 1) * 48 + (size_t)(K + 2) * 8 + (size_t)(K + 1) * 16 + (size_t)WORK_CAP * 4;
}

__host__ __device__ inline size_t kernel_smem_bytes(int W, int H, int K, int warps) {
    size_t b = (size_t)W * H * 8 + (size_t)warps * WARP_SMEM_BYTES + env_smem_bytes(K);
    return (b + 15) & ~(size_t)15;
}

// ------------------------------------------------------------------------------------------------
// K4: raster one triangle per lane (small) or per warp (big).  Called converged by the whole warp.
// ------------------------------------------------------------------------------------------------
template <bool STATS>
__device__ __forceinline__ void shade_px(const Edges &E, const float q[3], unsigned id2, int i, int j, int W,
                                         float zfar, unsigned long long *fb, unsigned &n_frag) {
    float f[3], num, depth;
    if (!cover_depth(E, q, i, j, f, num, depth)) return;
    if (STATS) ++n_frag;
    if (depth > zfar) return;
    const unsigned long long key = ((unsigned long long)__float_as_uint(depth) << 32) | id2;
    key_min(&fb[fb_index(i, j, W)], key);
}

template <bool STATS>
__device__ __forceinline__ void raster_warp(Tri &tri, bool have, int W, int H, float zfar, unsigned long long *fb,
                                            int lane, unsigned &n_tri, unsigned &n_frag) {
    int i0 = 0, i1 = -1, j0 = 0, j1 = -1;
    Edges E;
    bool big = false;
    if (have) have = pixel_bbox(tri.X, tri.Y, W, H, i0, i1, j0, j1);
    if (have) {
        long long A = area2(tri);
        if (A == 0) {
            have = false;
        } else {
            if (A < 0) { swap12(tri); A = -A; }
            edge_setup(tri, A, E);
        }
    }
    if (have) {
        if (STATS) ++n_tri;
        const int npx = (i1 - i0 + 1) * (j1 - j0 + 1);
        if (npx <= SMALL_MAX_PX) {
            for (int j = j0; j <= j1; ++j)
                for (int i = i0; i <= i1; ++i) shade_px<STATS>(E, tri.q, tri.id2, i, j, W, zfar, fb, n_frag);
        } else {
            big = true;
        }
    }
    unsigned mb = __ballot_sync(0xFFFFFFFFu, big);
    while (mb) {
        const int src = __ffs(mb) - 1;
        mb &= mb - 1;
        Tri bt;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            bt.X[k] = __shfl_sync(0xFFFFFFFFu, tri.X[k], src);
            bt.Y[k] = __shfl_sync(0xFFFFFFFFu, tri.Y[k], src);
            bt.q[k] = __shfl_sync(0xFFFFFFFFu, tri.q[k], src);
        }
        bt.id2 = __shfl_sync(0xFFFFFFFFu, tri.id2, src);
        int bi0, bi1, bj0, bj1;
        pixel_bbox(bt.X, bt.Y, W, H, bi0, bi1, bj0, bj1);
        Edges BE;
        edge_setup(bt, area2(bt), BE);   // the source lane already normalised the orientation: area > 0
        const int lx = lane & 7, ly = lane >> 3;
        for (int by = bj0 >> 2; by <= (bj1 >> 2); ++by)
            for (int bx = bi0 >> 3; bx <= (bi1 >> 3); ++bx)
                shade_px<STATS>(BE, bt.q, bt.id2, bx * 8 + lx, by * 4 + ly, W, zfar, fb, n_frag);
    }
}

// ------------------------------------------------------------------------------------------------
// N4 for one triangle: camera-space corners v[3] (+ optional colours) -> up to two clipped triangles.
// Returns the number of pieces; piece `sub` is written to o[3] (and oc).  COL = carry colours.
// ------------------------------------------------------------------------------------------------
template <bool COL>
__device__ __forceinline__ int clip_near(const CamVert v[3], const float c[3][3], float znear, int sub, CamVert o[3],
                                         float oc[3][3]) {
    const bool in0 = v[0].w >= znear, in1 = v[1].w >= znear, in2 = v[2].w >= znear;
    const int n_in = (int)in0 + (int)in1 + (int)in2;
    if (n_in == 0) return 0;
    if (n_in == 3) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            o[k] = v[k];
            if (COL) { oc[k][0] = c[k][0]; oc[k][1] = c[k][1]; oc[k][2] = c[k][2]; }
        }
        return 1;
    }
    // rotate: n_in == 1 -> a = the inside vertex; n_in == 2 -> c = the outside vertex, (a, b) follow it
    int k;
    if (n_in == 1) k = in0 ? 0 : (in1 ? 1 : 2);
    else k = !in0 ? 1 : (!in1 ? 2 : 0);   // index of a = (outside + 1) % 3
    CamVert r[3];
    float rc[3][3];
#pragma unroll
    for (int m = 0; m < 3; ++m) {
        const int src = (k + m) % 3;
        // (select written out so that the arrays stay in registers)
        r[m] = src == 0 ? v[0] : (src == 1 ? v[1] : v[2]);
        if (COL) {
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) rc[m][ch] = src == 0 ? c[0][ch] : (src == 1 ? c[1][ch] : c[2][ch]);
        }
    }
    // r = (a, b, c)
    auto P = [&](int in, int out, CamVert &p, float pc[3]) {
        const float t = clip_t(r[in].w, r[out].w, znear);
        p.xc = clip_lerp(t, r[in].xc, r[out].xc);
        p.yc = clip_lerp(t, r[in].yc, r[out].yc);
        p.w = znear;   // assigned, not interpolated
        if (COL) {
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) pc[ch] = clip_lerp(t, rc[in][ch], rc[out][ch]);
        }
    };
    if (n_in == 1) {   // (a, P(a,b), P(a,c))
        o[0] = r[0];
        if (COL) { oc[0][0] = rc[0][0]; oc[0][1] = rc[0][1]; oc[0][2] = rc[0][2]; }
        P(0, 1, o[1], oc[1]);
        P(0, 2, o[2], oc[2]);
        return 1;
    }
    // two inside, c outside: sub 0 = (a, b, P(b,c)), sub 1 = (a, P(b,c), P(a,c))
    o[0] = r[0];
    if (COL) { oc[0][0] = rc[0][0]; oc[0][1] = rc[0][1]; oc[0][2] = rc[0][2]; }
    if (sub == 0) {
        o[1] = r[1];
        if (COL) { oc[1][0] = rc[1][0]; oc[1][1] = rc[1][1]; oc[1][2] = rc[1][2]; }
        P(1, 2, o[2], oc[2]);
    } else {
        P(1, 2, o[1], oc[1]);
        P(0, 2, o[2], oc[2]);
    }
    return 2;
}

}  // namespace gx

namespace gx {

// ------------------------------------------------------------------------------------------------
// K2c: set-up of narrow survivors into the warp's record group.  Lanes [nrec, nrec + take) each set up one
// triangle of lst[g .. g + take); records [0, nrec) of earlier batches stay.  Returns take.
// ------------------------------------------------------------------------------------------------
template <bool STATS>
__device__ __forceinline__ int setup_fill(const WarpSmem &ws, const uchar4 *__restrict__ tris, uint32_t idb, int g,
                                          int nsurv, int nrec, int W, int H, int lane, unsigned &n_tri) {
    const int take = min(32 - nrec, nsurv - g);
    const int k = lane - nrec;
    if (k >= 0 && k < take) {
        const int t = ws.lst[g + k];
        const uchar4 ix = __ldg(&tris[t]);
        const int2 a = ws.vXY[ix.x], b = ws.vXY[ix.y], c = ws.vXY[ix.z];
        int X[3] = {a.x, b.x, c.x}, Y[3] = {a.y, b.y, c.y};
        float q[3] = {ws.vQ[ix.x], ws.vQ[ix.y], ws.vQ[ix.z]};
        int i0, i1, j0, j1;
        pixel_bbox(X, Y, W, H, i0, i1, j0, j1);   // non-empty: the triangle passed K2b
        // N6 in int32: |differences| < NARROW_EXT, so every product is < 2^30
        int A = (X[1] - X[0]) * (Y[2] - Y[0]) - (Y[1] - Y[0]) * (X[2] - X[0]);
        const bool degenerate = A == 0;
        if (A < 0) {
            A = -A;
            int ti = X[1]; X[1] = X[2]; X[2] = ti;
            ti = Y[1]; Y[1] = Y[2]; Y[2] = ti;
            const float tf = q[1]; q[1] = q[2]; q[2] = tf;
        }
        const int px0 = (i0 << 8) + 128, py0 = (j0 << 8) + 128;
        uint32_t bias_bits = 0;
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const int va = (e + 1) % 3, vb = (e + 2) % 3;
            int dx = X[vb] - X[va], dy = Y[vb] - Y[va];
            const bool tl = (dy < 0) || (dy == 0 && dx > 0);
            int E0 = dx * (py0 - Y[va]) - dy * (px0 - X[va]);
            if (degenerate) { E0 = -1; dx = 0; dy = 0; }   // covers nothing
            bias_bits |= (tl ? 0u : 1u) << e;
            ws.rec[(R_E0 + e) * 32 + lane] = (uint32_t)E0;
            ws.rec[(R_D0 + e) * 32 + lane] = ((uint32_t)dx << 16) | ((uint32_t)dy & 0xFFFFu);
            ws.rec[(R_Q0 + e) * 32 + lane] = __float_as_uint(q[e]);
        }
        ws.rec[R_FA * 32 + lane] = __float_as_uint((float)A);
        ws.rec[R_ID * 32 + lane] = (idb + (uint32_t)t) << 1;
        ws.rec[R_BB * 32 + lane] = (uint32_t)i0 | ((uint32_t)j0 << 7) | ((uint32_t)(i1 - i0) << 14) |
                                   ((uint32_t)(j1 - j0) << 21) | (bias_bits << 28);
        if (STATS) n_tri += degenerate ? 0u : 1u;
    }
    __syncwarp();
    return take;
}

// ------------------------------------------------------------------------------------------------
// K4b: depth (N7) and (depth, id) min (N9) for the queued fragments, one fragment per lane.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void shade_queue(const WarpSmem &ws, int qn, int W, float zfar, unsigned long long *fb,
                                            int lane) {
    for (int f = lane; f < qn; f += 32) {
        const uint32_t en = ws.fq[f];
        const int r = (int)(en & 31u), a = (int)((en >> 5) & 127u), b = (int)((en >> 12) & 127u);
        const uint32_t bb = ws.rec[R_BB * 32 + r];
        float fe[3], q[3];
#pragma unroll
        for (int e = 0; e < 3; ++e) {
            const uint32_t d = ws.rec[(R_D0 + e) * 32 + r];
            const int dx = (int)d >> 16, dy = (int)(short)(d & 0xFFFFu);
            const int Ee = (int)ws.rec[(R_E0 + e) * 32 + r] + ((b * dx - a * dy) << 8);
            fe[e] = (float)Ee;
            q[e] = __uint_as_float(ws.rec[(R_Q0 + e) * 32 + r]);
        }
        const float num = fmaf(fe[2], q[2], fmaf(fe[1], q[1], fe[0] * q[0]));
        const float depth = __uint_as_float(ws.rec[R_FA * 32 + r]) / num;
        if (depth > zfar) continue;
        const int x = (int)(bb & 127u) + a, y = (int)((bb >> 7) & 127u) + b;
        const unsigned long long key = ((unsigned long long)__float_as_uint(depth) << 32) | ws.rec[R_ID * 32 + r];
        key_min(&fb[fb_index(x, y, W)], key);
    }
    __syncwarp();
}

// ------------------------------------------------------------------------------------------------
// K3 + K4a: coverage of the nrec records of the warp's group.  The bounding boxes are cut into slots of 4
// pixels of one row; the T slots of the group are dealt to the lanes in equal contiguous runs (a lane walks
// through its run, moving to the next record when one is exhausted), so that lanes stay busy whatever the mix
// of triangle sizes.  Covered pixels are appended to the fragment queue and shaded densely by shade_queue.
// ------------------------------------------------------------------------------------------------
template <bool STATS>
__device__ __forceinline__ void raster_group(const WarpSmem &ws, int nrec, int W, float zfar, unsigned long long *fb,
                                             int lane, unsigned &n_frag) {
    const unsigned FULL = 0xFFFFFFFFu;
    int ns = 0;
    if (lane < nrec) {
        const uint32_t bb = ws.rec[R_BB * 32 + lane];
        const int w = (int)((bb >> 14) & 127u) + 1, h = (int)((bb >> 21) & 127u) + 1;
        ns = h * ((w + 3) >> 2);
    }
    int inc = ns;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(FULL, inc, d);
        if (lane >= d) inc += v;
    }
    const int T = __shfl_sync(FULL, inc, 31);
    const int Pex = inc - ns;
    const int per = (T + 31) >> 5;
    const int s0 = lane * per;
    const int n = min(per, T - s0);
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
        cw = (w + 3) >> 2;
    };
    load_rec(r);
    int row = off / cw, chunk = off - row * cw;
    int qn = 0;
    const uint32_t fq_addr = (uint32_t)__cvta_generic_to_shared(ws.fq);
    for (int it = 0; it < per; ++it) {
        const bool act = it < n;
        const int a = chunk << 2;
        unsigned m4 = 0;
        if (act) {
            int Ee[3], sx[3];
#pragma unroll
            for (int e = 0; e < 3; ++e) {
                Ee[e] = E0[e] + ((row * dx[e] - a * dy[e]) << 8);
                sx[e] = -(dy[e] << 8);
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const bool c = ((Ee[0] | Ee[1] | Ee[2]) >= 0) && (a + k < w);
                m4 |= (c ? 1u : 0u) << k;
                Ee[0] += sx[0]; Ee[1] += sx[1]; Ee[2] += sx[2];
            }
        }
        // append the covered pixels: one warp scan of the per-lane counts, then predicated stores
        const int cnt = __popc(m4);
        int incl = cnt;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int v = __shfl_up_sync(FULL, incl, d);
            if (lane >= d) incl += v;
        }
        const int tot = __shfl_sync(FULL, incl, 31);
        if (tot) {
            uint32_t en = (uint32_t)r | ((uint32_t)a << 5) | ((uint32_t)row << 12);
            uint32_t addr = fq_addr + (uint32_t)(qn + incl - cnt) * 4u;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
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
                    ++r;
                    if (it + 1 < n) load_rec(r);
                }
            }
        }
        if (qn > FQ_CAP - 128) {
            __syncwarp();
            if (STATS) n_frag += (lane == 0) ? (unsigned)qn : 0u;
            shade_queue(ws, qn, W, zfar, fb, lane);
            qn = 0;
        }
    }
    __syncwarp();
    if (qn) {
        if (STATS) n_frag += (lane == 0) ? (unsigned)qn : 0u;
        shade_queue(ws, qn, W, zfar, fb, lane);
    }
}

// ------------------------------------------------------------------------------------------------
// K2 + K3 + K4 for one batch, by one warp.  nrec (warp-uniform) = records pending in the warp's group.
// ------------------------------------------------------------------------------------------------
template <bool STATS>
__device__ __forceinline__ void process_batch(const GxParams &P, const Proj &pj, uint32_t item, const EnvSmem &es,
                                              const WarpSmem &ws, unsigned long long *fb, int lane, int &nrec,
                                              unsigned &n_in, unsigned &n_tri, unsigned &n_frag) {
    const uint32_t s = item >> 24;
    const GxBatchDev b = P.batches[item & 0xFFFFFFu];
    const int nv = (int)(b.nv_nt & 0xFFFFu), nt = (int)(b.nv_nt >> 16);
    float M[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) M[k] = es.MV[s * 12 + k];
    const uint32_t idb = es.id_base[s] + b.first_tri;
    const float4 *__restrict__ verts = P.verts + b.vert_off;
    const uchar4 *__restrict__ tris = P.tris + b.tri_off;
    const unsigned lt = (1u << lane) - 1u;
    if (STATS) n_in += (lane == 0) ? (unsigned)nt : 0u;

    // K2a: vertex transform, projection, snap -> warp-private staging
    for (int v = lane; v < nv; v += 32) {
        const float4 p = __ldg(&verts[v]);
        const CamVert cv = xform(M, p.x, p.y, p.z);
        int X = X_OUT, Y = 0;
        float q = 0.0f;
        if (cv.w >= P.znear) project(pj, cv.xc, cv.yc, cv.w, X, Y, q);
        ws.vXY[v] = make_int2(X, Y);
        ws.vQ[v] = q;
    }
    __syncwarp();

    // K2b: per triangle, near classification and the pixel-centre bounding-box reject; ballot-compact into
    // narrow survivors (front of lst) and slow-path triangles (back of lst)
    int nsurv = 0, nslow = 0;
    for (int t0 = 0; t0 < nt; t0 += 32) {
        const int t = t0 + lane;
        bool ok = false, slow = false;
        if (t < nt) {
            const uchar4 ix = __ldg(&tris[t]);
            const int2 a = ws.vXY[ix.x], bb = ws.vXY[ix.y], c = ws.vXY[ix.z];
            const int nout = (int)(a.x == X_OUT) + (int)(bb.x == X_OUT) + (int)(c.x == X_OUT);
            if (nout == 0) {
                const int X[3] = {a.x, bb.x, c.x}, Y[3] = {a.y, bb.y, c.y};
                int i0, i1, j0, j1;
                if (pixel_bbox(X, Y, P.W, P.H, i0, i1, j0, j1)) {
                    const int ext = max(max(X[0], max(X[1], X[2])) - min(X[0], min(X[1], X[2])),
                                        max(Y[0], max(Y[1], Y[2])) - min(Y[0], min(Y[1], Y[2])));
                    ok = ext < NARROW_EXT;
                    slow = !ok;
                }
            } else if (nout < 3) {
                slow = true;
            }
        }
        const unsigned mo = __ballot_sync(0xFFFFFFFFu, ok), mc = __ballot_sync(0xFFFFFFFFu, slow);
        if (ok) ws.lst[nsurv + __popc(mo & lt)] = (unsigned char)t;
        if (slow) ws.lst[255 - (nslow + __popc(mc & lt))] = (unsigned char)t;
        nsurv += __popc(mo);
        nslow += __popc(mc);
    }
    __syncwarp();

    // K2c + K3 + K4: narrow survivors through the record group
    for (int g = 0; g < nsurv;) {
        const int take = setup_fill<STATS>(ws, tris, idb, g, nsurv, nrec, P.W, P.H, lane, n_tri);
        g += take;
        nrec += take;
        if (nrec == 32) {
            raster_group<STATS>(ws, 32, P.W, P.zfar, fb, lane, n_frag);
            nrec = 0;
        }
    }

    // slow path: wide triangles (int64 edge functions) and near-plane straddlers (N4 clip), piece by piece
    for (int g = 0; g < nslow; g += 32) {
        const bool have = g + lane < nslow;
        CamVert cv[3];
        Tri whole;
        int t = 0;
        bool clipped = false;
        if (have) {
            t = ws.lst[255 - (g + lane)];
            const uchar4 ix = __ldg(&tris[t]);
            const int2 a = ws.vXY[ix.x], bb = ws.vXY[ix.y], c = ws.vXY[ix.z];
            clipped = a.x == X_OUT || bb.x == X_OUT || c.x == X_OUT;
            if (clipped) {
                const float4 p0 = __ldg(&verts[ix.x]), p1 = __ldg(&verts[ix.y]), p2 = __ldg(&verts[ix.z]);
                cv[0] = xform(M, p0.x, p0.y, p0.z);
                cv[1] = xform(M, p1.x, p1.y, p1.z);
                cv[2] = xform(M, p2.x, p2.y, p2.z);
            } else {
                whole.X[0] = a.x; whole.X[1] = bb.x; whole.X[2] = c.x;
                whole.Y[0] = a.y; whole.Y[1] = bb.y; whole.Y[2] = c.y;
                whole.q[0] = ws.vQ[ix.x]; whole.q[1] = ws.vQ[ix.y]; whole.q[2] = ws.vQ[ix.z];
            }
        }
#pragma unroll 1
        for (int sub = 0; sub < 2; ++sub) {
            Tri tri;
            bool h2 = false;
            if (have) {
                if (clipped) {
                    CamVert o[3];
                    const int np = clip_near<false>(cv, nullptr, P.znear, sub, o, nullptr);
                    h2 = sub < np;
                    if (h2) {
#pragma unroll
                        for (int k = 0; k < 3; ++k) project(pj, o[k].xc, o[k].yc, o[k].w, tri.X[k], tri.Y[k], tri.q[k]);
                    }
                } else {
                    h2 = sub == 0;
                    tri = whole;
                }
                tri.id2 = ((idb + (uint32_t)t) << 1) | (unsigned)sub;
            }
            raster_warp<STATS>(tri, h2, P.W, P.H, P.zfar, fb, lane, n_tri, n_frag);
        }
    }
    __syncwarp();
}

// ------------------------------------------------------------------------------------------------
// K5a: colour of the winning triangle at pixel (i, j), recomputed from the mesh (N8).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t resolve_color(const GxParams &P, const Proj &pj, const EnvSmem &es, unsigned id2,
                                                  int i, int j) {
    const uint32_t id = id2 >> 1;
    const int sub = (int)(id2 & 1u);
    int lo = 0, hi = P.K;
    while (lo < hi) {   // largest slot whose first id is <= id (empty slots never win: they own no id)
        const int mid = (lo + hi + 1) >> 1;
        if (es.id_base[mid] <= id) lo = mid; else hi = mid - 1;
    }
    const int s = lo;
    const uint32_t tl = id - es.id_base[s];
    const GxClusterDev cl = P.clusters[es.slot_cl[s] + (tl >> 8)];
    GxBatchDev b = P.batches[cl.batch_off];
    for (uint32_t bi = 1; bi < cl.nbatch && tl - b.first_tri >= (b.nv_nt >> 16); ++bi) b = P.batches[cl.batch_off + bi];
    const uchar4 ix = __ldg(&P.tris[b.tri_off + (tl - b.first_tri)]);
    const float4 p[3] = {__ldg(&P.verts[b.vert_off + ix.x]), __ldg(&P.verts[b.vert_off + ix.y]),
                         __ldg(&P.verts[b.vert_off + ix.z])};
    float M[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) M[k] = es.MV[s * 12 + k];
    CamVert cv[3], o[3];
    float c[3][3], oc[3][3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        cv[k] = xform(M, p[k].x, p[k].y, p[k].z);
        const uint32_t rgba = __float_as_uint(p[k].w);
        c[k][0] = (float)(rgba & 0xFFu);
        c[k][1] = (float)((rgba >> 8) & 0xFFu);
        c[k][2] = (float)((rgba >> 16) & 0xFFu);
    }
    clip_near<true>(cv, c, P.znear, sub, o, oc);
    Tri tri;
#pragma unroll
    for (int k = 0; k < 3; ++k) project(pj, o[k].xc, o[k].yc, o[k].w, tri.X[k], tri.Y[k], tri.q[k]);
    long long A = area2(tri);
    if (A < 0) {
        swap12(tri);
        A = -A;
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) { const float f = oc[1][ch]; oc[1][ch] = oc[2][ch]; oc[2][ch] = f; }
    }
    Edges E;
    edge_setup(tri, A, E);
    float f[3], num, depth;
    cover_depth(E, tri.q, i, j, f, num, depth);   // covered by construction: this triangle won the pixel
    uint32_t out = 0;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
        const float g0 = tri.q[0] * oc[0][ch], g1 = tri.q[1] * oc[1][ch], g2 = tri.q[2] * oc[2][ch];
        const float cn = fmaf(f[2], g2, fmaf(f[1], g1, f[0] * g0));
        const float v = cn / num;
        out |= (uint32_t)fminf(255.0f, fmaxf(0.0f, rintf(v))) << (8 * ch);
    }
    return out;
}

}  // namespace gx

namespace gx {

// ------------------------------------------------------------------------------------------------
// K1: conservative frustum test of one cluster AABB under model-view M (K1).
// The object-space box is mapped to a camera-space box (centre MV*c, half extent |MV3x3|*e, inflated),
// which contains every vertex of the cluster and every vertex N4 can create (those lie on segments
// between vertices).  The cluster is skipped only if the whole box is behind the near plane, beyond the
// far plane, or outside one of the four side planes |fx*xc| <= w, |fy*yc| <= w; outside a side plane every
// snapped X is <= 0 or >= 256*W (resp. Y), half a pixel away from the nearest pixel centre, which dwarfs
// the float32 error of the box arithmetic (margin m below).
// ------------------------------------------------------------------------------------------------
// camera-space box of a cluster: centre, inflated half extents, margin m, depth range
struct CamBox { float cx, cy, ex, ey, m, wmin, wmax; };

__device__ __forceinline__ CamBox cluster_box(const GxClusterDev &c, const float *M) {
    const float hx = 0.5f * (c.bmax[0] - c.bmin[0]), hy = 0.5f * (c.bmax[1] - c.bmin[1]),
                hz = 0.5f * (c.bmax[2] - c.bmin[2]);
    const float ox = 0.5f * (c.bmax[0] + c.bmin[0]), oy = 0.5f * (c.bmax[1] + c.bmin[1]),
                oz = 0.5f * (c.bmax[2] + c.bmin[2]);
    const float cx = M[0] * ox + M[1] * oy + M[2] * oz + M[3];
    const float cy = M[4] * ox + M[5] * oy + M[6] * oz + M[7];
    const float cz = M[8] * ox + M[9] * oy + M[10] * oz + M[11];
    float ex = fabsf(M[0]) * hx + fabsf(M[1]) * hy + fabsf(M[2]) * hz;
    float ey = fabsf(M[4]) * hx + fabsf(M[5]) * hy + fabsf(M[6]) * hz;
    float ez = fabsf(M[8]) * hx + fabsf(M[9]) * hy + fabsf(M[10]) * hz;
    // margin: 1e-4 relative to every magnitude that entered the sums (float32 error is ~1e-6 of that)
    const float mag = fabsf(M[0] * ox) + fabsf(M[1] * oy) + fabsf(M[2] * oz) + fabsf(M[3]) + fabsf(M[4] * ox) +
                      fabsf(M[5] * oy) + fabsf(M[6] * oz) + fabsf(M[7]) + fabsf(M[8] * ox) + fabsf(M[9] * oy) +
                      fabsf(M[10] * oz) + fabsf(M[11]) + ex + ey + ez;
    CamBox b;
    b.m = 1e-4f * mag + 1e-5f;
    b.cx = cx; b.cy = cy;
    b.ex = ex + b.m; b.ey = ey + b.m;
    ez += b.m;
    b.wmax = -cz + ez;
    b.wmin = -cz - ez;
    return b;
}

__device__ __forceinline__ bool box_in_frustum(const CamBox &b, float fx, float fy, float znear, float zfar) {
    const float m = b.m;
    if (b.wmax < znear) return false;                     // every vertex fails w >= znear
    if (b.wmin > zfar * 1.0001f + m) return false;        // every fragment has depth > zfar
    if (fx * (b.cx - b.ex) - b.wmax > m) return false;    // right of the image
    if (-fx * (b.cx + b.ex) - b.wmax > m) return false;   // left
    if (fy * (b.cy - b.ey) - b.wmax > m) return false;    // above
    if (-fy * (b.cy + b.ey) - b.wmax > m) return false;   // below
    return true;
}

__device__ __forceinline__ bool cluster_visible(const GxClusterDev &c, const float *M, float fx, float fy, float znear,
                                                float zfar) {
    return box_in_frustum(cluster_box(c, M), fx, fy, znear, zfar);
}


// ------------------------------------------------------------------------------------------------
// per-environment setup by the whole CTA (two barriers inside): slot tables, model-view matrices (N1, N2),
// exclusive scans of triangle and cluster counts over the K+1 slots.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void env_setup(const GxParams &P, int env, const EnvSmem &es, int tid) {
    const int K = P.K, lane = tid & 31, warp = tid >> 5;
    for (int sl = tid; sl <= K; sl += (int)blockDim.x) {
        int mesh = -1;
        if (sl == 0) mesh = P.env_scene[env];
        else {
            const int m = P.inst_mesh[(size_t)env * K + (sl - 1)];
            if (m >= 0) mesh = P.n_static + m;
        }
        uint32_t nt = 0, nc = 0, cl0 = 0;
        if (mesh >= 0) {
            const GxMeshDev md = P.meshes[mesh];
            nt = md.nt; nc = md.ncluster; cl0 = md.cluster_off;
        }
        es.slot_mesh[sl] = mesh; es.slot_nt[sl] = nt; es.slot_nc[sl] = nc; es.slot_cl[sl] = cl0;
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
// K1 for the clusters [c0, c1) of the environment's cluster space, by the whole CTA: survivors' batches are
// appended to es.work by warp-aggregated shared atomics (*s_work_n must be 0 and visible on entry; the
// caller synchronises afterwards).
// ------------------------------------------------------------------------------------------------
template <bool STATS>
__device__ __forceinline__ void cull_chunk_to_worklist(const GxParams &P, const EnvSmem &es, uint32_t c0, uint32_t c1,
                                                       int tid, int NT, unsigned *s_work_n, unsigned &st_tested,
                                                       unsigned &st_drawn) {
    const int K = P.K, lane = tid & 31, warp = tid >> 5;
    for (uint32_t g0 = c0 + warp * 32; g0 < c1; g0 += NT) {
        const uint32_t g = g0 + lane;
        uint32_t nb = 0, boff = 0, s = 0;
        if (g < c1) {
            int lo = 0, hi = K;
            while (lo < hi) {   // largest slot whose first cluster index is <= g
                const int mid = (lo + hi + 1) >> 1;
                if (es.cl_base[mid] <= g) lo = mid; else hi = mid - 1;
            }
            s = (uint32_t)lo;
            const GxClusterDev c = P.clusters[es.slot_cl[s] + (g - es.cl_base[s])];
            const bool vis = !P.cull || cluster_visible(c, es.MV + s * 12, P.fx, P.fy, P.znear, P.zfar);
            if (STATS) { ++st_tested; st_drawn += vis ? 1u : 0u; }
            if (vis) { nb = c.nbatch; boff = c.batch_off; }
        }
        uint32_t inc = nb;   // warp-aggregated append: one shared atomic per warp
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t a = __shfl_up_sync(0xFFFFFFFFu, inc, d);
            if (lane >= d) inc += a;
        }
        const uint32_t tot = __shfl_sync(0xFFFFFFFFu, inc, 31);
        uint32_t base = 0;
        if (lane == 0 && tot) base = atomicAdd(s_work_n, tot);
        base = __shfl_sync(0xFFFFFFFFu, base, 0) + inc - nb;
        for (uint32_t k = 0; k < nb; ++k) es.work[base + k] = (s << 24) | (boff + k);
    }
}

// ------------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------------
template <int WARPS, int MINB, bool STATS>
__global__ void __launch_bounds__(WARPS * 32, MINB) render_kernel(const GxParams P) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NT = WARPS * 32;
    const int W = P.W, H = P.H, K = P.K, npix = W * H;

    unsigned long long *fb = reinterpret_cast<unsigned long long *>(smem);
    unsigned char *p = smem + (size_t)npix * 8;
    WarpSmem ws;
    {
        unsigned char *w = p + (size_t)warp * WARP_SMEM_BYTES;
        ws.vXY = reinterpret_cast<int2 *>(w);
        ws.vQ = reinterpret_cast<float *>(w + GX_VCAP * 8);
        ws.lst = w + GX_VCAP * 12;
        ws.rec = reinterpret_cast<uint32_t *>(w + GX_VCAP * 12 + 256);
        ws.fq = ws.rec + REC_WORDS * 32;
    }
    p += (size_t)WARPS * WARP_SMEM_BYTES;
    EnvSmem es;
    es.MV = reinterpret_cast<float *>(p);          p += (size_t)(K + 1) * 48;
    es.id_base = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 2) * 4;
    es.cl_base = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 2) * 4;
    es.slot_cl = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 1) * 4;
    es.slot_mesh = reinterpret_cast<int32_t *>(p); p += (size_t)(K + 1) * 4;
    es.slot_nt = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 1) * 4;
    es.slot_nc = reinterpret_cast<uint32_t *>(p);  p += (size_t)(K + 1) * 4;
    es.work = reinterpret_cast<uint32_t *>(p);

    __shared__ int s_env;
    __shared__ unsigned s_work_n, s_work_next;
    __shared__ unsigned long long s_stat[GX_NSTAT];

    Proj pj;
    pj.fx = P.fx; pj.fy = P.fy;
    pj.hw = 128.0f * (float)W; pj.hh = 128.0f * (float)H;

    unsigned st_tested = 0, st_drawn = 0, st_in = 0, st_tri = 0, st_frag = 0;
    if (STATS) {
        if (tid < GX_NSTAT) s_stat[tid] = 0;
    }

    for (;;) {
        if (tid == 0) s_env = (int)atomicAdd(P.env_counter, 1u);
        __syncthreads();
        const int env = s_env;
        if (env >= P.N) break;
        if (P.env_filter && !P.env_filter[env]) {   // overflow pass of the two-kernel path: flagged environments only
            __syncthreads();
            continue;
        }

        // ---- environment setup: clear the frame; slots, model-view matrices (N1, N2), id / cluster bases ----
        {
            uint4 *f4 = reinterpret_cast<uint4 *>(fb);
            const uint4 ones = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
            for (int k = tid; k < npix / 2; k += NT) f4[k] = ones;
        }
        env_setup(P, env, es, tid);

        // ---- K1 cull + K2..K4 draw, in chunks of the environment's cluster space -------------------
        const uint32_t n_cl = es.cl_base[K + 1];
        int nrec = 0;
        for (uint32_t c0 = 0; c0 < n_cl; c0 += (uint32_t)P.cull_chunk) {
            if (tid == 0) { s_work_n = 0; s_work_next = 0; }
            __syncthreads();
            cull_chunk_to_worklist<STATS>(P, es, c0, min(c0 + (uint32_t)P.cull_chunk, n_cl), tid, NT, &s_work_n, st_tested, st_drawn);
            __syncthreads();
            const unsigned n_work = s_work_n;
            for (;;) {
                unsigned wi = 0;
                if (lane == 0) wi = atomicAdd(&s_work_next, 1u);
                wi = __shfl_sync(0xFFFFFFFFu, wi, 0);
                if (wi >= n_work) break;
                process_batch<STATS>(P, pj, es.work[wi], es, ws, fb, lane, nrec, st_in, st_tri, st_frag);
            }
            __syncthreads();
        }
        if (nrec) {   // records still pending in this warp's group
            raster_group<STATS>(ws, nrec, W, P.zfar, fb, lane, st_frag);
            nrec = 0;
        }
        __syncthreads();

        // ---- K5a: resolve in place: key -> (depth bits, rgba) ------------------------------------
        const bool want_rgb = P.rgb != nullptr || P.obs != nullptr;
        for (int k = tid; k < npix; k += NT) {
            const int j = k / W, i = k - j * W;       // row-linear order: coalesced id stores
            const int a = fb_index(i, j, W);
            const unsigned long long key = fb[a];
            uint32_t dbits = 0, rgba = 0, id = 0xFFFFFFFFu;
            if (key != KEY_BG) {
                dbits = (uint32_t)(key >> 32);
                id = (uint32_t)key >> 1;
                if (want_rgb) rgba = resolve_color(P, pj, es, (uint32_t)key, i, j);
            }
            fb[a] = ((unsigned long long)rgba << 32) | dbits;
            if (P.id) P.id[(size_t)env * npix + k] = id;
        }
        __syncthreads();

        // ---- K5b: write out, 4 pixels per thread, 16-byte stores -----------------------------------
        for (int k = tid; k < npix / 4; k += NT) {
            const int pix = k * 4;
            const int j = pix / W, i = pix - j * W;
            const int a = fb_index(i, j, W);          // 4-aligned columns stay contiguous under the XOR
            const uint4 v0 = *reinterpret_cast<const uint4 *>(&fb[a]);
            const uint4 v1 = *reinterpret_cast<const uint4 *>(&fb[a + 2]);
            float4 d;
            d.x = __uint_as_float(v0.x); d.y = __uint_as_float(v0.z);
            d.z = __uint_as_float(v1.x); d.w = __uint_as_float(v1.z);
            if (P.depth) *reinterpret_cast<float4 *>(P.depth + (size_t)env * npix + pix) = d;
            if (P.obs) {
                const uint32_t oc[4] = {v0.y, v0.w, v1.y, v1.w};
                const float od[4] = {d.x, d.y, d.z, d.w};
                store_obs4(P.obs + (size_t)env * 4 * npix, (size_t)npix, (size_t)pix, oc, od, P.obs_dmin, P.obs_range);
            }
            if (P.rgb) {
                // 4 pixels = 12 bytes = 3 words per lane; 4 lanes hold 48 bytes = three 16-byte stores
                const uint32_t c0 = v0.y, c1 = v0.w, c2 = v1.y, c3 = v1.w;
                const uint32_t w0 = (c0 & 0xFFFFFFu) | (c1 << 24);
                const uint32_t w1 = ((c1 >> 8) & 0xFFFFu) | (c2 << 16);
                const uint32_t w2 = ((c2 >> 16) & 0xFFu) | (c3 << 8);
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
                    uint8_t *dst = P.rgb + ((size_t)env * npix + (size_t)(pix - 4 * g)) * 3 + 16 * g;
                    *reinterpret_cast<uint4 *>(dst) = make_uint4(o[0], o[1], o[2], o[3]);
                }
            }
        }
        __syncthreads();
    }

    if (STATS) {
        atomicAdd(&s_stat[GX_STAT_CLUSTERS_TESTED], (unsigned long long)st_tested);
        atomicAdd(&s_stat[GX_STAT_CLUSTERS_DRAWN], (unsigned long long)st_drawn);
        atomicAdd(&s_stat[GX_STAT_TRIS_IN], (unsigned long long)st_in);
        atomicAdd(&s_stat[GX_STAT_TRIS_RASTER], (unsigned long long)st_tri);
        atomicAdd(&s_stat[GX_STAT_FRAGMENTS], (unsigned long long)st_frag);
        __syncthreads();
        if (tid < GX_NSTAT) atomicAdd(&P.stats[tid], s_stat[tid]);
    }
}

}  // namespace gx
