/*
 * gx_oracle.c -- the CPU ORACLE of the batch RGBD rasteriser.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
 * load or call this file.  It shares no code, header, table or helper with the CUDA path under
 * paper_2306_07552_b200/csrc/ and includes nothing from include/.
 *
 * What it computes.  The paper states the problem only (section 3.1: one renderer
 * instance renders all environments, shared assets, per-step scene-graph updates in, one stack of
 * images per sensor out; section 4.1: 128x128 RGBD, 90-degree FoV head camera) and is
 * silent on every numerical detail of rasterisation.  The per-pixel definition is therefore the
 * reading N0..N10 listed in DESIGN.md section 3 (taken from SURVEY.md section 8(c) and
 * BASELINE.json north_star: 8-bit sub-pixel fixed point, integer edge functions, top-left fill rule,
 * lowest-triangle-id tie break, barycentric uint8 vertex colours, float32 linear depth):
 *
 *   for every environment and every pixel, among all post-clip, post-snap triangles of that
 *   environment whose integer edge functions cover the pixel centre under the top-left rule and whose
 *   interpolated depth is <= zfar, the one with the lexicographically smallest (depth, id, sub);
 *   output its depth and interpolated colour, or the background.
 *
 * It is that plain definition written out: a loop over environments, over all triangles, over the
 * pixels of the triangle's bounding box.  No culling, no tiling, no SIMD, no reordering.  All
 * floating point is IEEE-754 binary32, round-to-nearest-even, built with -ffp-contract=off; fmaf()
 * appears exactly where the definition says fma.
 *
 * Pins (tests/test_oracle_pins.py, `-m "not gpu"`): closed-form vertex positions (N1-N5), closed-form
 * axis-aligned quads and exact big-integer brute force of the perturbed-sample definition of the
 * top-left rule (N6), watertight-grid invariant (N6), near-clip invariants (N4), exact power-of-two
 * depth and double-precision ray casting (N7), constant / affine colour closed forms and
 * double-precision ray casting (N8), order/id permutation invariants (N9), full-scan == bbox (N6).
 * Parity unpinned: exact RGB value where perspective correction matters beyond +-1 LSB of the
 * double-precision ray caster.
 *
 * Also here (end of the file): N11, the packed float16 observation, and N12, the scene-graph update (forward
 * kinematics of the robot, Table 5) that produces the camera and link transforms
 * the renderer reads.  N12 pins: its own sine / cosine against float64 and the exact values at 0; closed forms
 * (joints at 0 with dyadic offsets, a quarter turn about each axis, a prismatic joint, base yaw); random
 * chains against a float64 composition; parent / child and held-object identities.
 * And N13, the batch collision queries of the kinematic simulator (spheres against column grids and oriented boxes,
 * PAPER.md:111-119, App. G): pins in tests/test_collide_pins.py (closed forms, boundary cases, float64 brute force).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    const float *positions;  /* [nv*3] */
    const uint8_t *colors;   /* [nv*3] RGB */
    const uint32_t *indices; /* [nt*3] */
    uint32_t nv, nt;
} OrMesh;

typedef struct {
    int32_t width, height;
    float fx, fy; /* NDC focal lengths: fy = 1/tan(fovy/2), fx = fy*H/W */
    float znear, zfar;
} OrCamera;

/* camera-space vertex after N3: position (xc, yc), w = -zc, colour as 3 floats */
typedef struct {
    float xc, yc, w, c[3];
} OrVert;

typedef struct {
    const OrCamera *cam;
    float *dstar;     /* [H*W] best depth so far, +inf = none   (N9) */
    uint32_t *idstar; /* [H*W] */
    uint8_t *substar; /* [H*W] */
    uint8_t *rgb;     /* [H*W*3] */
    uint32_t *count;  /* [H*W] or NULL: number of covering fragments, depth test ignored */
    int full_scan;    /* 1: visit every pixel instead of the bounding box */
} OrTarget;

#define OR_BACKGROUND_ID 0xFFFFFFFFu

/* N1: view matrix from the rigid camera-to-world pose C (row-major 4x4).
 * V[i][j] = C[j][i] (exact transpose), V[i][3] = -fma(C[2][i],C[2][3], fma(C[1][i],C[1][3], C[0][i]*C[0][3])). */
static void or_view_matrix(const float *C, float V[3][4]) {
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) V[i][j] = C[j * 4 + i];
        V[i][3] = -fmaf(C[2 * 4 + i], C[2 * 4 + 3], fmaf(C[1 * 4 + i], C[1 * 4 + 3], C[0 * 4 + i] * C[0 * 4 + 3]));
    }
}

/* N2: model-view.  Static mesh: MV = V.  Instance with M = top 3 rows of inst_xform. */
static void or_model_view(const float V[3][4], const float *M /* 16 floats or NULL */, float MV[3][4]) {
    if (!M) {
        memcpy(MV, V, sizeof(float) * 12);
        return;
    }
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j)
            MV[i][j] = fmaf(V[i][2], M[2 * 4 + j], fmaf(V[i][1], M[1 * 4 + j], V[i][0] * M[0 * 4 + j]));
        MV[i][3] = fmaf(V[i][2], M[2 * 4 + 3], fmaf(V[i][1], M[1 * 4 + 3], fmaf(V[i][0], M[0 * 4 + 3], V[i][3])));
    }
}

/* N3: camera-space vertex.  The camera looks along -Z, so w = -zc. */
static OrVert or_vertex(const float MV[3][4], const float *p, const uint8_t *col) {
    OrVert v;
    float x = p[0], y = p[1], z = p[2];
    v.xc = fmaf(MV[0][2], z, fmaf(MV[0][1], y, fmaf(MV[0][0], x, MV[0][3])));
    v.yc = fmaf(MV[1][2], z, fmaf(MV[1][1], y, fmaf(MV[1][0], x, MV[1][3])));
    float zc = fmaf(MV[2][2], z, fmaf(MV[2][1], y, fmaf(MV[2][0], x, MV[2][3])));
    v.w = -zc;
    v.c[0] = (float)col[0];
    v.c[1] = (float)col[1];
    v.c[2] = (float)col[2];
    return v;
}

/* N4: the new vertex on the edge from an inside vertex to an outside vertex, at w = znear.
 * Always computed from the inside vertex towards the outside vertex, so both triangles sharing a
 * clipped edge get the identical vertex. */
static OrVert or_clip_point(const OrVert *in, const OrVert *out, float znear) {
    OrVert p;
    float t = (in->w - znear) / (in->w - out->w);
    p.xc = fmaf(t, out->xc - in->xc, in->xc);
    p.yc = fmaf(t, out->yc - in->yc, in->yc);
    for (int k = 0; k < 3; ++k) p.c[k] = fmaf(t, out->c[k] - in->c[k], in->c[k]);
    p.w = znear; /* assigned, not interpolated */
    return p;
}

/* N5..N9 for one post-clip triangle. */
static void or_raster_clipped(OrTarget *T, const OrVert tri[3], uint32_t id, uint8_t sub) {
    const OrCamera *cam = T->cam;
    const int W = cam->width, H = cam->height;
    const float hw = 128.0f * (float)W, hh = 128.0f * (float)H; /* exact */
    const float LIM = 268435456.0f;                               /* 2^28 */
    int32_t X[3], Y[3];
    float q[3], c[3][3];
    /* N5: projection and snap to 1/256 pixel, round-half-even */
    for (int k = 0; k < 3; ++k) {
        q[k] = 1.0f / tri[k].w;
        float Xf = fmaf((cam->fx * tri[k].xc) * q[k], hw, hw);
        float Yf = fmaf(-((cam->fy * tri[k].yc) * q[k]), hh, hh);
        Xf = fminf(fmaxf(Xf, -LIM), LIM);
        Yf = fminf(fmaxf(Yf, -LIM), LIM);
        X[k] = (int32_t)rintf(Xf);
        Y[k] = (int32_t)rintf(Yf);
        for (int ch = 0; ch < 3; ++ch) c[k][ch] = tri[k].c[ch];
    }
    /* N6: signed doubled area, orientation normalisation, no back-face culling */
    int64_t A = (int64_t)(X[1] - X[0]) * (int64_t)(Y[2] - Y[0]) - (int64_t)(Y[1] - Y[0]) * (int64_t)(X[2] - X[0]);
    if (A == 0) return;
    if (A < 0) {
        int32_t ti;
        float tf;
        ti = X[1]; X[1] = X[2]; X[2] = ti;
        ti = Y[1]; Y[1] = Y[2]; Y[2] = ti;
        tf = q[1]; q[1] = q[2]; q[2] = tf;
        for (int ch = 0; ch < 3; ++ch) { tf = c[1][ch]; c[1][ch] = c[2][ch]; c[2][ch] = tf; }
        A = -A;
    }
    /* edge e runs from a = v[(e+1)%3] to b = v[(e+2)%3]; E_e weights vertex e */
    int64_t dx[3], dy[3];
    int32_t Xa[3], Ya[3];
    int topleft[3];
    for (int e = 0; e < 3; ++e) {
        int a = (e + 1) % 3, b = (e + 2) % 3;
        Xa[e] = X[a];
        Ya[e] = Y[a];
        dx[e] = (int64_t)X[b] - (int64_t)X[a];
        dy[e] = (int64_t)Y[b] - (int64_t)Y[a];
        topleft[e] = (dy[e] < 0) || (dy[e] == 0 && dx[e] > 0);
    }
    /* pixel bounding box (exact: contains every pixel centre inside the vertex bounding box) */
    int imin = 0, imax = W - 1, jmin = 0, jmax = H - 1;
    if (!T->full_scan) {
        int32_t Xmin = X[0] < X[1] ? X[0] : X[1]; if (X[2] < Xmin) Xmin = X[2];
        int32_t Xmax = X[0] > X[1] ? X[0] : X[1]; if (X[2] > Xmax) Xmax = X[2];
        int32_t Ymin = Y[0] < Y[1] ? Y[0] : Y[1]; if (Y[2] < Ymin) Ymin = Y[2];
        int32_t Ymax = Y[0] > Y[1] ? Y[0] : Y[1]; if (Y[2] > Ymax) Ymax = Y[2];
        /* floor division by 256 written out (no reliance on arithmetic shifts of negatives) */
        int64_t a0 = (int64_t)Xmin + 127, a1 = (int64_t)Xmax - 128, b0 = (int64_t)Ymin + 127, b1 = (int64_t)Ymax - 128;
        int64_t i0 = a0 >= 0 ? a0 / 256 : -((-a0 + 255) / 256);
        int64_t i1 = a1 >= 0 ? a1 / 256 : -((-a1 + 255) / 256);
        int64_t j0 = b0 >= 0 ? b0 / 256 : -((-b0 + 255) / 256);
        int64_t j1 = b1 >= 0 ? b1 / 256 : -((-b1 + 255) / 256);
        if (i0 > imin) imin = (int)(i0 > W ? W : i0);
        if (i1 < imax) imax = (int)(i1 < -1 ? -1 : i1);
        if (j0 > jmin) jmin = (int)(j0 > H ? H : j0);
        if (j1 < jmax) jmax = (int)(j1 < -1 ? -1 : j1);
    }
    const float fA = (float)A;
    for (int j = jmin; j <= jmax; ++j) {
        for (int i = imin; i <= imax; ++i) {
            const int64_t px = 256 * (int64_t)i + 128, py = 256 * (int64_t)j + 128; /* pixel centre */
            int64_t E[3];
            int covered = 1;
            for (int e = 0; e < 3; ++e) {
                E[e] = dx[e] * (py - Ya[e]) - dy[e] * (px - Xa[e]);
                if (!(E[e] > 0 || (E[e] == 0 && topleft[e]))) covered = 0;
            }
            if (!covered) continue;
            const size_t p = (size_t)j * (size_t)W + (size_t)i;
            if (T->count) T->count[p] += 1;
            /* N7: planar view-space depth, perspective-correct */
            float f0 = (float)E[0], f1 = (float)E[1], f2 = (float)E[2];
            float num = fmaf(f2, q[2], fmaf(f1, q[1], f0 * q[0]));
            float depth = fA / num;
            if (depth > cam->zfar) continue;
            /* N9: (depth, id, sub) lexicographic minimum */
            float ds = T->dstar[p];
            int wins = (depth < ds) ||
                       (depth == ds && (id < T->idstar[p] || (id == T->idstar[p] && sub < T->substar[p])));
            if (!wins) continue;
            T->dstar[p] = depth;
            T->idstar[p] = id;
            T->substar[p] = sub;
            /* N8: perspective-correct colour, shares num */
            for (int ch = 0; ch < 3; ++ch) {
                float g0 = q[0] * c[0][ch], g1 = q[1] * c[1][ch], g2 = q[2] * c[2][ch];
                float cn = fmaf(f2, g2, fmaf(f1, g1, f0 * g0));
                float v = cn / num;
                T->rgb[p * 3 + ch] = (uint8_t)fminf(255.0f, fmaxf(0.0f, rintf(v)));
            }
        }
    }
}

/* N4: near-plane clip of one camera-space triangle, then N5..N9 for each piece. */
static void or_raster_triangle(OrTarget *T, const OrVert v[3], uint32_t id) {
    const float znear = T->cam->znear;
    int in[3], n_in = 0;
    for (int k = 0; k < 3; ++k) {
        in[k] = v[k].w >= znear;
        n_in += in[k];
    }
    if (n_in == 0) return;
    if (n_in == 3) {
        or_raster_clipped(T, v, id, 0);
        return;
    }
    if (n_in == 1) {
        int k = in[0] ? 0 : (in[1] ? 1 : 2);
        const OrVert *a = &v[k], *b = &v[(k + 1) % 3], *c = &v[(k + 2) % 3]; /* a inside */
        OrVert t[3] = {*a, or_clip_point(a, b, znear), or_clip_point(a, c, znear)};
        or_raster_clipped(T, t, id, 0);
        return;
    }
    { /* two inside: rotate so that c is the outside vertex */
        int k = !in[0] ? 0 : (!in[1] ? 1 : 2);
        const OrVert *c = &v[k], *a = &v[(k + 1) % 3], *b = &v[(k + 2) % 3];
        OrVert pbc = or_clip_point(b, c, znear), pac = or_clip_point(a, c, znear);
        OrVert t0[3] = {*a, *b, pbc};
        OrVert t1[3] = {*a, pbc, pac};
        or_raster_clipped(T, t0, id, 0);
        or_raster_clipped(T, t1, id, 1);
    }
}

static void or_target_begin(OrTarget *T, size_t npix) {
    for (size_t p = 0; p < npix; ++p) {
        T->dstar[p] = INFINITY;
        T->idstar[p] = OR_BACKGROUND_ID;
        T->substar[p] = 0;
        T->rgb[3 * p] = T->rgb[3 * p + 1] = T->rgb[3 * p + 2] = 0;
        if (T->count) T->count[p] = 0;
    }
}

/* N9 background: rgb (0,0,0) (already), depth 0.0f, id 0xFFFFFFFF */
static void or_target_end(OrTarget *T, size_t npix, float *depth_out) {
    for (size_t p = 0; p < npix; ++p) depth_out[p] = (T->idstar[p] == OR_BACKGROUND_ID) ? 0.0f : T->dstar[p];
}

static int or_camera_ok(const OrCamera *c) {
    return c && c->width > 0 && c->height > 0 && c->znear > 0.0f && c->zfar > c->znear;
}

/* ---------------------------------------------------------------------------------------------
 * exported entry points
 * ------------------------------------------------------------------------------------------- */

/* Whole definition for a batch: environments are independent, so the loop over them
 * may run on several threads; nothing else is parallel.  rgb [N,H,W,3] u8, depth [N,H,W] f32,
 * id [N,H,W] u32; sub [N,H,W] u8 and count [N,H,W] u32 may be NULL.  Returns 0, or -1 on bad args. */
int gx_oracle_render(const OrMesh *static_meshes, int32_t n_static, const OrMesh *dyn_meshes, int32_t n_dyn,
                     const OrCamera *cam, int32_t N, int32_t K, const int32_t *env_scene, const float *cam_pose,
                     const int32_t *inst_mesh, const float *inst_xform, uint8_t *rgb, float *depth, uint32_t *id,
                     uint8_t *sub, uint32_t *count, int32_t flags, int32_t n_threads) {
    if (!or_camera_ok(cam) || N < 0 || K < 0 || !rgb || !depth || !id || n_static <= 0) return -1;
    const size_t npix = (size_t)cam->width * (size_t)cam->height;
    for (int n = 0; n < N; ++n) {
        if (env_scene[n] < 0 || env_scene[n] >= n_static) return -1;
        for (int k = 0; k < K; ++k)
            if (inst_mesh[(size_t)n * K + k] >= n_dyn) return -1;
    }
    if (n_threads < 1) n_threads = 1;
    int err = 0;
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
    for (int n = 0; n < N; ++n) {
        uint8_t *sub_local = sub ? sub + (size_t)n * npix : (uint8_t *)malloc(npix);
        float *dstar = (float *)malloc(npix * sizeof(float));
        if (!sub_local || !dstar) {
            err = 1;
            free(dstar);
            if (!sub) free(sub_local);
            continue;
        }
        OrTarget T = {cam, dstar, id + (size_t)n * npix, sub_local, rgb + (size_t)n * npix * 3,
                      count ? count + (size_t)n * npix : NULL, flags & 1};
        or_target_begin(&T, npix);
        float V[3][4], MV[3][4];
        or_view_matrix(cam_pose + (size_t)n * 16, V);
        /* triangle id: static triangle j -> j; triangle j of instance slot k ->
         * T_static + sum of nt over earlier non-empty slots + j */
        uint32_t id_base = 0;
        for (int slot = -1; slot < K; ++slot) {
            const OrMesh *m;
            const float *M = NULL;
            if (slot < 0) {
                m = &static_meshes[env_scene[n]];
            } else {
                int32_t mi = inst_mesh[(size_t)n * K + slot];
                if (mi < 0) continue;
                m = &dyn_meshes[mi];
                M = inst_xform + ((size_t)n * K + slot) * 16;
            }
            or_model_view(V, M, MV);
            for (uint32_t j = 0; j < m->nt; ++j) {
                OrVert v[3];
                for (int c = 0; c < 3; ++c) {
                    uint32_t vi = m->indices[3 * (size_t)j + c];
                    v[c] = or_vertex(MV, m->positions + 3 * (size_t)vi, m->colors + 3 * (size_t)vi);
                }
                or_raster_triangle(&T, v, id_base + j);
            }
            id_base += m->nt;
        }
        or_target_end(&T, npix, depth + (size_t)n * npix);
        free(dstar);
        if (!sub) free(sub_local);
    }
    return err ? -2 : 0;
}

/* N4..N9 on an explicit camera-space triangle soup: verts [nt][3][6] = (xc, yc, w, r, g, b) per
 * corner, ids [nt].  Triangles are processed in array order; by N9 the result must not depend on it. */
int gx_oracle_raster_soup(const OrCamera *cam, const float *verts, const uint32_t *ids, uint32_t nt, uint8_t *rgb,
                          float *depth, uint32_t *id, uint8_t *sub, uint32_t *count, int32_t flags) {
    if (!or_camera_ok(cam) || !rgb || !depth || !id) return -1;
    const size_t npix = (size_t)cam->width * (size_t)cam->height;
    uint8_t *sub_local = sub ? sub : (uint8_t *)malloc(npix);
    float *dstar = (float *)malloc(npix * sizeof(float));
    if (!sub_local || !dstar) return -2;
    OrTarget T = {cam, dstar, id, sub_local, rgb, count, flags & 1};
    or_target_begin(&T, npix);
    for (uint32_t t = 0; t < nt; ++t) {
        OrVert v[3];
        for (int c = 0; c < 3; ++c) {
            const float *s = verts + ((size_t)t * 3 + c) * 6;
            v[c].xc = s[0]; v[c].yc = s[1]; v[c].w = s[2];
            v[c].c[0] = s[3]; v[c].c[1] = s[4]; v[c].c[2] = s[5];
        }
        or_raster_triangle(&T, v, ids[t]);
    }
    or_target_end(&T, npix, depth);
    free(dstar);
    if (!sub) free(sub_local);
    return 0;
}

/* N1..N3 + N5 for a vertex array (no clipping): camera-space (xc, yc, w), inside flag (w >= znear),
 * and for inside vertices q = 1/w and the snapped (Xi, Yi).  xform may be NULL (static mesh). */
int gx_oracle_vertex_stage(const OrCamera *cam, const float *cam_pose, const float *xform, const float *positions,
                           uint32_t nv, float *xc, float *yc, float *w, float *q, int32_t *Xi, int32_t *Yi,
                           uint8_t *inside) {
    if (!or_camera_ok(cam)) return -1;
    float V[3][4], MV[3][4];
    const uint8_t black[3] = {0, 0, 0};
    or_view_matrix(cam_pose, V);
    or_model_view(V, xform, MV);
    const float hw = 128.0f * (float)cam->width, hh = 128.0f * (float)cam->height, LIM = 268435456.0f;
    for (uint32_t i = 0; i < nv; ++i) {
        OrVert v = or_vertex(MV, positions + 3 * (size_t)i, black);
        xc[i] = v.xc; yc[i] = v.yc; w[i] = v.w;
        inside[i] = v.w >= cam->znear;
        q[i] = 0.0f; Xi[i] = 0; Yi[i] = 0;
        if (inside[i]) {
            q[i] = 1.0f / v.w;
            float Xf = fmaf((cam->fx * v.xc) * q[i], hw, hw);
            float Yf = fmaf(-((cam->fy * v.yc) * q[i]), hh, hh);
            Xi[i] = (int32_t)rintf(fminf(fmaxf(Xf, -LIM), LIM));
            Yi[i] = (int32_t)rintf(fminf(fmaxf(Yf, -LIM), LIM));
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * N11 (NEXT-1 of SURVEY.md 8(f)): the packed observation the policy reads (PAPER.md:91,
 * PAPER.md:141 "RGBD").  The paper is silent on layout and normalisation; the reading is
 *   out[n][0..2][y][x] = binary16( (float)c / 255.0f ),  c = uint8 channel of the rendered image
 *   out[n][3][y][x]    = binary16( (clamp(depth, dmin, dmax) - dmin) / (dmax - dmin) )
 * all operations IEEE binary32, conversions round-to-nearest-even.
 * or_half_rn: binary32 -> binary16 bits, written out by hand (non-negative finite inputs): normal, subnormal,
 * ties to even, overflow to infinity.
 * ------------------------------------------------------------------------------------------------ */
static uint16_t or_half_rn(float f) {
    uint32_t x;
    memcpy(&x, &f, 4);
    const uint32_t sign = (x >> 16) & 0x8000u;
    const int exp = (int)((x >> 23) & 0xFFu);
    uint32_t man = x & 0x7FFFFFu;
    if (exp == 0xFF) return (uint16_t)(sign | 0x7C00u | (man ? 0x200u : 0u));
    if (exp == 0) return (uint16_t)sign;                 /* binary32 subnormal: far below half of the smallest binary16 */
    const int e = exp - 127 + 15;
    if (e >= 31) return (uint16_t)(sign | 0x7C00u);
    if (e <= 0) {                                        /* binary16 subnormal: value = man16 * 2^-24 */
        if (e < -10) return (uint16_t)sign;
        man |= 0x800000u;
        const int shift = 14 - e;                        /* 14 .. 24 */
        uint32_t h = man >> shift;
        const uint32_t rem = man & ((1u << shift) - 1u), half = 1u << (shift - 1);
        if (rem > half || (rem == half && (h & 1u))) ++h;
        return (uint16_t)(sign | h);
    }
    uint32_t h = ((uint32_t)e << 10) | (man >> 13);
    const uint32_t rem = man & 0x1FFFu;
    if (rem > 0x1000u || (rem == 0x1000u && (h & 1u))) ++h;   /* a carry into the exponent is the right answer */
    return (uint16_t)(sign | h);
}

int gx_oracle_pack_obs(const uint8_t *rgb /* [N,H,W,3] */, const float *depth /* [N,H,W] */, int32_t N, int32_t H,
                       int32_t W, float dmin, float dmax, uint16_t *out /* [N,4,H,W] */) {
    if (!rgb || !depth || !out || N <= 0 || H <= 0 || W <= 0 || !(dmax > dmin)) return -1;
    const size_t npix = (size_t)H * (size_t)W;
    const float range = dmax - dmin;
    for (int32_t n = 0; n < N; ++n)
        for (size_t p = 0; p < npix; ++p) {
            for (int ch = 0; ch < 3; ++ch) {
                const float v = (float)rgb[((size_t)n * npix + p) * 3 + ch] / 255.0f;
                out[((size_t)n * 4 + ch) * npix + p] = or_half_rn(v);
            }
            float d = depth[(size_t)n * npix + p];
            d = fminf(fmaxf(d, dmin), dmax);
            out[((size_t)n * 4 + 3) * npix + p] = or_half_rn((d - dmin) / range);
        }
    return 0;
}

/* binary32 -> binary16 of an array: exposes or_half_rn to its pins */
void gx_oracle_half_rn(const float *in, uint16_t *out, size_t n) {
    for (size_t k = 0; k < n; ++k) out[k] = or_half_rn(in[k]);
}

/* ------------------------------------------------------------------------------------------------
 * N12: scene-graph update -- forward kinematics from base pose and joint positions to the link, camera and
 * held-object transforms the renderer reads (N12; "we use forward kinematics
 * to compute the position of the robot's articulated links", "Scene graph updates are communicated
 * ... to the ... renderer", Table 5 PAPER.md:416 "Render Setup").  Plain loops, one environment after the
 * other, link after link in index order (a parent always has a smaller index than its child).
 * All operations are IEEE binary32; fmaf is the single-rounding fused multiply-add; nothing is contracted.
 * ------------------------------------------------------------------------------------------------ */

/* N12a: sine and cosine in binary32: Cody-Waite reduction by multiples of pi/2 in two steps, then the degree-7 /
 * degree-8 polynomials on [-pi/4, pi/4] evaluated by Horner's rule with fmaf, then the quadrant. */
static void n12_sincos(float x, float *s_out, float *c_out) {
    const float k = rintf(x * 0.636619772f);               /* nearest multiple of pi/2 */
    float r = fmaf(-k, 1.57079625f, x);                    /* pi/2 = 1.57079625 + 7.54978942e-08 (+ ...) */
    r = fmaf(-k, 7.54978942e-08f, r);
    const float z = r * r;
    float ps = fmaf(z, -1.9515295891e-4f, 8.3321608736e-3f);
    ps = fmaf(z, ps, -1.6666654611e-1f);
    const float sn = fmaf(r * z, ps, r);                   /* sin r */
    float pc = fmaf(z, 2.443315711809948e-5f, -1.388731625493765e-3f);
    pc = fmaf(z, pc, 4.166664568298827e-2f);
    const float cs = fmaf(z * z, pc, fmaf(-0.5f, z, 1.0f)); /* cos r */
    const int q = (int)k & 3;                              /* two's complement: also right for negative k */
    float s = (q & 1) ? cs : sn, c = (q & 1) ? sn : cs;
    if (q == 1 || q == 2) c = -c;
    if (q >= 2) s = -s;
    *s_out = s;
    *c_out = c;
}

/* affine product C = A * B of two 3x4 matrices (rows of 4, implicit last row 0 0 0 1), the operation order of N2 */
static void n12_mul(const float *A, const float *B, float *C) {
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j)
            C[i * 4 + j] = fmaf(A[i * 4 + 2], B[8 + j], fmaf(A[i * 4 + 1], B[4 + j], A[i * 4] * B[j]));
        C[i * 4 + 3] = fmaf(A[i * 4 + 2], B[11], fmaf(A[i * 4 + 1], B[7], fmaf(A[i * 4], B[3], A[i * 4 + 3])));
    }
}

/* N12b: joint transform.  type 0 fixed: identity; 1 revolute about the unit axis a by theta (Rodrigues);
 * 2 prismatic along a by theta. */
static void n12_joint(int type, const float *a, float theta, float *J) {
    for (int k = 0; k < 12; ++k) J[k] = (k % 5 == 0) ? 1.0f : 0.0f;
    if (type == 1) {
        float s, c;
        n12_sincos(theta, &s, &c);
        const float t = 1.0f - c;
        J[0] = fmaf(t * a[0], a[0], c);
        J[1] = fmaf(t * a[0], a[1], -(s * a[2]));
        J[2] = fmaf(t * a[0], a[2], s * a[1]);
        J[4] = fmaf(t * a[1], a[0], s * a[2]);
        J[5] = fmaf(t * a[1], a[1], c);
        J[6] = fmaf(t * a[1], a[2], -(s * a[0]));
        J[8] = fmaf(t * a[2], a[0], -(s * a[1]));
        J[9] = fmaf(t * a[2], a[1], s * a[0]);
        J[10] = fmaf(t * a[2], a[2], c);
    } else if (type == 2) {
        J[3] = theta * a[0];
        J[7] = theta * a[1];
        J[11] = theta * a[2];
    }
}

typedef struct {
    int32_t parent;      /* index of the parent link, -1 = the base */
    int32_t joint_type;  /* 0 fixed, 1 revolute, 2 prismatic */
    float axis[3];       /* unit joint axis in the joint frame */
    float origin[12];    /* 3x4: joint frame in the parent link's frame */
} GxOracleLink;

static void n12_store44(float *dst, const float *M) {
    for (int k = 0; k < 12; ++k) dst[k] = M[k];
    dst[12] = 0.0f; dst[13] = 0.0f; dst[14] = 0.0f; dst[15] = 1.0f;
}

/* N12c.  base_pose [N,3] = (x, z, yaw): the base stands on the ground plane y = 0 and turns about +Y.
 * W_base = Ry(yaw) with translation (x, 0, z); W_l = W_parent(l) * (origin_l * J_l(joint_pos[n][l])).
 * Writes inst_xform[n][link_slot0 + l] = W_l (4x4 row-major), cam_pose[n] = W_camera_link * cam_mount, and, where
 * held_slot[n] >= 0, inst_xform[n][held_slot[n]] = W_ee_link * held_xform[n].  Other slots are left alone.
 * Returns 0, or -1 on bad arguments. */
int gx_oracle_fk(const GxOracleLink *links, int32_t L, int32_t camera_link, const float *cam_mount /* [12] */, int32_t ee_link,
                 int32_t N, int32_t K, int32_t link_slot0, const float *base_pose, const float *joint_pos /* [N,L] */,
                 const int32_t *held_slot /* [N] or NULL */, const float *held_xform /* [N,12] or NULL */,
                 float *cam_pose /* [N,16] */, float *inst_xform /* [N,K,16] */) {
    if (!links || L <= 0 || L > 64 || N <= 0 || !base_pose || !joint_pos || !cam_pose || !cam_mount) return -1;
    if (camera_link < -1 || camera_link >= L || ee_link < -1 || ee_link >= L) return -1;
    if (link_slot0 < 0 || link_slot0 + L > K || (K > 0 && !inst_xform)) return -1;
    for (int l = 0; l < L; ++l)
        if (links[l].parent < -1 || links[l].parent >= l) return -1;
    for (int n = 0; n < N; ++n) {
        float W[65][12];   /* W[0] = base, W[l + 1] = link l */
        float s, c;
        n12_sincos(base_pose[3 * n + 2], &s, &c);
        const float B[12] = {c, 0.0f, s, base_pose[3 * n], 0.0f, 1.0f, 0.0f, 0.0f, -s, 0.0f, c, base_pose[3 * n + 1]};
        for (int k = 0; k < 12; ++k) W[0][k] = B[k];
        for (int l = 0; l < L; ++l) {
            float J[12], Loc[12];
            n12_joint(links[l].joint_type, links[l].axis, joint_pos[(size_t)n * L + l], J);
            n12_mul(links[l].origin, J, Loc);
            n12_mul(W[links[l].parent + 1], Loc, W[l + 1]);
            n12_store44(inst_xform + ((size_t)n * K + link_slot0 + l) * 16, W[l + 1]);
        }
        float Cm[12];
        n12_mul(W[camera_link + 1], cam_mount, Cm);
        n12_store44(cam_pose + (size_t)n * 16, Cm);
        if (held_slot && held_xform && held_slot[n] >= 0) {
            if (held_slot[n] >= K) return -1;
            float Hm[12];
            n12_mul(W[ee_link + 1], held_xform + (size_t)n * 12, Hm);
            n12_store44(inst_xform + ((size_t)n * K + held_slot[n]) * 16, Hm);
        }
    }
    return 0;
}

/* N12a alone, for its pins */
void gx_oracle_sincos(const float *x, float *s, float *c, size_t n) {
    for (size_t i = 0; i < n; ++i) n12_sincos(x[i], &s[i], &c[i]);
}

/* ------------------------------------------------------------------------------------------------
 * N13: batch collision queries of the kinematic simulator (N13; PAPER.md:111-119 and
 * Appendix G): every sphere of the robot against the static scene's column grid of its radius
 * and against the oriented boxes of the resting movable objects.  The paper's regular grids and its layer cache
 * are accelerations that do not change the answer, so the oracle is the plain definition: nearest column, linear
 * search of its layers from the first; every object, one after the other.  All operations binary32.
 * ------------------------------------------------------------------------------------------------ */
typedef struct {
    float x0, z0;            /* world position of column (0, 0) */
    float spacing;           /* 0.03 m in the paper */
    int32_t nx, nz;
    const uint32_t *col_off; /* [nx*nz + 1] first layer of column iz*nx + ix */
    const float *layers;     /* [..][2] lo, hi: free heights of the sphere CENTRE (the radius is baked in) */
} GxOracleColumnGrid;

typedef struct {
    int32_t link;            /* link the sphere is attached to (>= 0) */
    int32_t radius_class;    /* index into radii[] */
    float centre[3];         /* in the link's frame (link == -1: in the grasped object's frame) */
} GxOracleSphere;

/* object-space box of a mesh: centre 0.5f*(min+max), half extent 0.5f*(max-min) of its vertex positions */
static void n13_mesh_box(const OrMesh *m, float *ctr, float *half) {
    float lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    for (uint32_t v = 0; v < m->nv; ++v)
        for (int a = 0; a < 3; ++a) {
            const float p = m->positions[3 * (size_t)v + a];
            if (v == 0 || p < lo[a]) lo[a] = p;
            if (v == 0 || p > hi[a]) hi[a] = p;
        }
    for (int a = 0; a < 3; ++a) { ctr[a] = 0.5f * (lo[a] + hi[a]); half[a] = 0.5f * (hi[a] - lo[a]); }
}

/* out_static[n][s] = 1 if sphere s of environment n is in obstructed space of its column grid (or outside the grid),
 * out_object[n][s] = lowest instance slot in [obj_slot0, obj_slot0 + n_obj) whose box the sphere overlaps (distance
 * from the centre to the box <= radius), skipping empty slots and held_slot[n]; -1 if none.
 * grids: [n_static][n_radii].  Sphere centres: W_link * centre with W_link = inst_xform[n][link_slot0 + link].
 * Returns 0, or -1 on bad arguments. */
int gx_oracle_collide(const OrMesh *dyn_meshes, int32_t n_dyn, const GxOracleColumnGrid *grids, int32_t n_static,
                      int32_t n_radii, const float *radii, const GxOracleSphere *spheres, int32_t S, int32_t N, int32_t K,
                      const int32_t *env_scene, const int32_t *inst_mesh, const float *inst_xform, int32_t link_slot0,
                      int32_t obj_slot0, int32_t n_obj, const int32_t *held_slot /* [N] or NULL */, uint8_t *out_static,
                      int32_t *out_object) {
    if (!grids || !radii || !spheres || S <= 0 || N <= 0 || !env_scene || !inst_xform || !out_static || !out_object) return -1;
    if (obj_slot0 < 0 || n_obj < 0 || obj_slot0 + n_obj > K || (n_obj > 0 && (!inst_mesh || !dyn_meshes))) return -1;
    for (int n = 0; n < N; ++n) {
        if (env_scene[n] < 0 || env_scene[n] >= n_static) return -1;
        for (int s = 0; s < S; ++s) {
            const GxOracleSphere *sp = &spheres[s];
            if (sp->link < -1 || (sp->link >= 0 && link_slot0 + sp->link >= K) || sp->radius_class < 0 || sp->radius_class >= n_radii) return -1;
            /* "we approximate the robot (and the current grasped object, if any) with a set of spheres"
             * (PAPER.md:111): link == -1 attaches the sphere to the grasped object -- its centre is given in that
             * object's frame and moves with inst_xform[n][held_slot[n]].  With nothing in the gripper the sphere does
             * not exist: it reports free space and no object. */
            int frame = link_slot0 + sp->link;
            if (sp->link == -1) {
                const int hs = held_slot ? held_slot[n] : -1;
                if (hs >= K) return -1;
                if (hs < 0) {
                    out_static[(size_t)n * S + s] = 0;
                    out_object[(size_t)n * S + s] = -1;
                    continue;
                }
                frame = hs;
            }
            const float *Wl = inst_xform + ((size_t)n * K + frame) * 16;
            float c[3];
            for (int i = 0; i < 3; ++i)   /* N3's order */
                c[i] = fmaf(Wl[i * 4 + 2], sp->centre[2], fmaf(Wl[i * 4 + 1], sp->centre[1], fmaf(Wl[i * 4], sp->centre[0], Wl[i * 4 + 3])));
            /* static scene: nearest column, then its layers */
            const GxOracleColumnGrid *g = &grids[(size_t)env_scene[n] * n_radii + sp->radius_class];
            const float fx = rintf((c[0] - g->x0) / g->spacing), fz = rintf((c[2] - g->z0) / g->spacing);
            int hit = 1;
            if (fx >= 0.0f && fx < (float)g->nx && fz >= 0.0f && fz < (float)g->nz) {
                const size_t col = (size_t)(int)fz * g->nx + (size_t)(int)fx;
                for (uint32_t l = g->col_off[col]; l < g->col_off[col + 1]; ++l)
                    if (g->layers[2 * (size_t)l] <= c[1] && c[1] <= g->layers[2 * (size_t)l + 1]) { hit = 0; break; }
            }
            out_static[(size_t)n * S + s] = (uint8_t)hit;
            /* resting movable objects: every slot, lowest overlapping one */
            const float r = radii[sp->radius_class], r2 = r * r;
            int found = -1;
            for (int k = obj_slot0; k < obj_slot0 + n_obj && found < 0; ++k) {
                const int mesh = inst_mesh[(size_t)n * K + k];
                if (mesh < 0 || (held_slot && held_slot[n] == k)) continue;
                if (mesh >= n_dyn) return -1;
                float bc[3], bh[3];
                n13_mesh_box(&dyn_meshes[mesh], bc, bh);
                const float *M = inst_xform + ((size_t)n * K + k) * 16;
                const float d[3] = {c[0] - M[3], c[1] - M[7], c[2] - M[11]};
                float e[3];
                for (int i = 0; i < 3; ++i) {
                    const float loc = fmaf(M[8 + i], d[2], fmaf(M[4 + i], d[1], M[i] * d[0]));   /* R^T d */
                    const float rel = loc - bc[i];
                    const float q = fminf(fmaxf(rel, -bh[i]), bh[i]);
                    e[i] = rel - q;
                }
                const float dist2 = fmaf(e[2], e[2], fmaf(e[1], e[1], e[0] * e[0]));
                if (dist2 <= r2) found = k;
            }
            out_object[(size_t)n * S + s] = found;
        }
    }
    return 0;
}
