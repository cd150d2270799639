// gx_math.cuh -- device functions shared by the stages of the render path (sm_100a): the arithmetic of DESIGN.md
// section 3 (N1-N9, N11) operation by operation, the conservative cluster-box tests of K1, and the per-environment
// slot tables.  Compiled with -fmad=false so that only the fmaf() calls written here fuse.
// Product code: nothing here is shared with oracle/.
#pragma once
#include <cuda_fp16.h>
#include "gx_types.h"

namespace gx {

constexpr unsigned long long KEY_BG = 0xFFFFFFFFFFFFFFFFull;
constexpr int X_OUT = (int)0x80000000;   // staged X of a vertex behind the near plane
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


// N11: packed policy observation of 4 consecutive pixels of one row: planes R, G, B =
// binary16(c / 255.0f), plane D = binary16((clamp(depth, dmin, dmax) - dmin) / range); all float32
// operations, round-to-nearest-even conversions.  obs points at plane 0 of the environment, pix = y * W + x.
__device__ __forceinline__ void store_obs4(uint16_t *obs, size_t npix, size_t pix, const uint32_t col[4], const float d[4],
                                           float dmin, float dmax, float range) {
#pragma unroll
    for (int ch = 0; ch < 4; ++ch) {
        unsigned short h[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            float v;
            if (ch < 3) v = (float)((col[m] >> (8 * ch)) & 0xFFu) / 255.0f;
            else v = (fminf(fmaxf(d[m], dmin), dmax) - dmin) / range;
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

// Occluder class of a sub-cluster (32 triangles) in the occluder scheme: big on screen (screen box of at least
// occl_area pixels per triangle) or reaching the near plane -- many pixels for little geometry.  Any
// classification gives the same image; this one only decides what can be culled.
__device__ __forceinline__ bool sub_is_occluder(const CamBox &b, float fx, float fy, int W, int H, float znear, float occl_area) {
    if (!(b.wmin >= znear)) return true;
    const float iw = 1.0f / b.wmin;   // the nearest depth gives the largest possible screen box
    const float wpx = fminf(2.0f * b.ex * fx * iw * 0.5f * (float)W, (float)W);
    const float hpx = fminf(2.0f * b.ey * fy * iw * 0.5f * (float)H, (float)H);
    return wpx * hpx >= occl_area * 32.0f;
}

// Occlusion test of a sub-cluster's camera-space box against the hi-Z pyramid of the occluder phase (hz: bits of
// the largest stored depth per 16x16-pixel tile, 0xFFFFFFFF where background shows; then the same per 2x2 tiles,
// 4x4 tiles, ... level after level): true only if every fragment the box can produce is strictly behind what is
// already drawn at every pixel it can touch, so that it can never win N9 and the image stays bit-identical (N10).
// The level is the finest one at which the box's pixel range spans at most 2x2 entries.
template <bool COOP>
__device__ __forceinline__ bool box_occluded(const CamBox &b, const uint32_t *hz, int tiles_x, int tiles_y, float fx, float fy,
                                             int W, int H, float znear) {
    if (!(b.wmin >= znear)) return false;   // reaches the near plane: no screen bound
    const float xl = b.cx - b.ex, xh = b.cx + b.ex, yl = b.cy - b.ey, yh = b.cy + b.ey;
    const float iw0 = 1.0f / b.wmin, iw1 = 1.0f / b.wmax;
    const float nxl = fx * xl * (xl >= 0.0f ? iw1 : iw0), nxh = fx * xh * (xh >= 0.0f ? iw0 : iw1);
    const float nyl = fy * yl * (yl >= 0.0f ? iw1 : iw0), nyh = fy * yh * (yh >= 0.0f ? iw0 : iw1);
    // pixel range, padded by one pixel for the 1/256 snap and the float error of the box arithmetic
    const float fW = (float)W, fH = (float)H;
    int tx0 = (int)fminf(fmaxf(floorf((nxl * 0.5f + 0.5f) * fW) - 1.0f, 0.0f), fW - 1.0f) >> 4;
    int tx1 = (int)fminf(fmaxf(floorf((nxh * 0.5f + 0.5f) * fW) + 1.0f, 0.0f), fW - 1.0f) >> 4;
    int ty0 = (int)fminf(fmaxf(floorf((-nyh * 0.5f + 0.5f) * fH) - 1.0f, 0.0f), fH - 1.0f) >> 4;
    int ty1 = (int)fminf(fmaxf(floorf((-nyl * 0.5f + 0.5f) * fH) + 1.0f, 0.0f), fH - 1.0f) >> 4;
    int off = 0, w = tiles_x, h = tiles_y;
    while (tx1 - tx0 > 1 || ty1 - ty0 > 1) {
        off += w * h;
        w = (w + 1) >> 1; h = (h + 1) >> 1;
        tx0 >>= 1; tx1 >>= 1; ty0 >>= 1; ty1 >>= 1;
    }
    const uint32_t *p = hz + off;
    const int a00 = ty0 * w + tx0, a01 = ty0 * w + tx1, a10 = ty1 * w + tx0, a11 = ty1 * w + tx1;
    const uint32_t zb = COOP ? max(max(__ldcg(&p[a00]), __ldcg(&p[a01])), max(__ldcg(&p[a10]), __ldcg(&p[a11])))
                             : max(max(__ldg(&p[a00]), __ldg(&p[a01])), max(__ldg(&p[a10]), __ldg(&p[a11])));
    return b.wmin * (1.0f - 1e-4f) > __uint_as_float(zb);   // (background: NaN, the comparison is false)
}

__device__ __forceinline__ bool cluster_visible(const GxClusterDev &c, const float *M, float fx, float fy, float znear,
                                                float zfar) {
    return box_in_frustum(cluster_box(c, M), fx, fy, znear, zfar);
}

}  // namespace gx
