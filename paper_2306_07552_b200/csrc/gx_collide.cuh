// gx_collide.cuh -- the batch collision queries of gx_collide_batch (sm_100a): every sphere of the robot against the
// static scene's column grid of its radius and against the oriented boxes of the resting movable objects (DESIGN.md
// section 3, N13; PAPER.md:111-119 and Appendix G).  The paper's layer cache and its four offset
// regular grids are CPU accelerations of the same answer; here an environment's boxes sit in shared memory and every
// sphere tests all of them.  Arithmetic follows N13 operation by operation (-fmad=false: only the fmaf() calls fuse).
// Product code: nothing here is shared with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace gx {

struct ColGridDev {          // one (static scene, radius class) column grid
    float x0, z0, spacing;
    int32_t nx, nz;
    uint32_t col_base;       // first entry of this grid in col_off (its nx*nz + 1 entries)
    uint32_t layer_base;     // first layer of this grid in layers
    uint32_t pad;
};

struct SphereDev { int32_t link, radius_class; float cx, cy, cz; };   // link == -1: rides on the grasped object (slot held_slot[n])

struct CollideParams {
    const ColGridDev *grids;     // [n_static * n_radii]
    const uint32_t *col_off;     // concatenated, relative to the grid's layer_base
    const float2 *layers;        // concatenated (lo, hi)
    const float *radii;          // [n_radii]
    const SphereDev *spheres;    // [S]
    const float4 *mesh_box;      // [n_dyn][2]: (centre, 0), (half extent, 0) of the mesh's object-space box
    int32_t n_static, n_radii, n_dyn, S;
    int32_t N, K, link_slot0, obj_slot0, n_obj;
    const int32_t *env_scene;
    const int32_t *inst_mesh;
    const float *inst_xform;
    const int32_t *held_slot;    // [N] or NULL
    uint8_t *out_static;         // [N,S]
    int32_t *out_object;         // [N,S]
};

constexpr int COLLIDE_MAX_OBJ = 64;      // resting objects per environment staged in shared memory at a time

// One warp per environment; lane = sphere (in rounds of 32).  The environment's object boxes (inverse rotation rows,
// translation, box centre and half extent) are staged in shared memory once, in rounds of COLLIDE_MAX_OBJ slots.
template <int WARPS>
__global__ void __launch_bounds__(WARPS * 32) collide_kernel(const CollideParams P) {
    __shared__ float s_obj[WARPS][COLLIDE_MAX_OBJ][20];   // M rows 0..2 (12), centre (3), half (3), valid, pad
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = blockIdx.x * WARPS + warp;
    if (n >= P.N) return;
    const int scene = P.env_scene[n];
    const int held = P.held_slot ? P.held_slot[n] : -1;
    const float *xf = P.inst_xform + (size_t)n * P.K * 16;
    for (int s0 = 0; s0 < P.S; s0 += 32) {
        const int s = s0 + lane;
        const bool have = s < P.S;
        float cx = 0.f, cy = 0.f, cz = 0.f, r2 = 0.f;
        int hit = 1;
        bool active = have;      // a sphere of the grasped object (link == -1) exists only while something is held
        if (have) {
            const SphereDev sp0 = P.spheres[s];
            if (sp0.link < 0) active = held >= 0 && held < P.K;
            if (!active) hit = 0;
        }
        if (active) {
            const SphereDev sp = P.spheres[s];
            const float *W = xf + (size_t)(sp.link < 0 ? held : P.link_slot0 + sp.link) * 16;
            cx = fmaf(W[2], sp.cz, fmaf(W[1], sp.cy, fmaf(W[0], sp.cx, W[3])));      // N3's order
            cy = fmaf(W[6], sp.cz, fmaf(W[5], sp.cy, fmaf(W[4], sp.cx, W[7])));
            cz = fmaf(W[10], sp.cz, fmaf(W[9], sp.cy, fmaf(W[8], sp.cx, W[11])));
            const float r = P.radii[sp.radius_class];
            r2 = r * r;
            // static scene: nearest column of the grid of this radius, then its layers
            if (scene >= 0 && scene < P.n_static) {
                const ColGridDev g = P.grids[(size_t)scene * P.n_radii + sp.radius_class];
                const float fx = rintf((cx - g.x0) / g.spacing), fz = rintf((cz - g.z0) / g.spacing);
                if (fx >= 0.0f && fx < (float)g.nx && fz >= 0.0f && fz < (float)g.nz) {
                    const uint32_t *off = P.col_off + g.col_base + (size_t)(int)fz * g.nx + (size_t)(int)fx;
                    const uint32_t l0 = off[0], l1 = off[1];
                    const float2 *lay = P.layers + g.layer_base;
                    for (uint32_t l = l0; l < l1; ++l) {
                        const float2 v = lay[l];
                        if (v.x <= cy && cy <= v.y) { hit = 0; break; }
                    }
                }
            }
        }
        // resting movable objects, lowest overlapping slot
        int found = -1;
        for (int k0 = 0; k0 < P.n_obj; k0 += COLLIDE_MAX_OBJ) {
            const int nk = min(COLLIDE_MAX_OBJ, P.n_obj - k0);
            __syncwarp();
            for (int k = lane; k < nk; k += 32) {
                const int slot = P.obj_slot0 + k0 + k;
                const int mesh = P.inst_mesh[(size_t)n * P.K + slot];
                const bool valid = mesh >= 0 && mesh < P.n_dyn && slot != held;
                float *o = s_obj[warp][k];
                o[18] = valid ? 1.0f : 0.0f;
                if (valid) {
                    const float4 *M = reinterpret_cast<const float4 *>(xf + (size_t)slot * 16);
                    const float4 m0 = M[0], m1 = M[1], m2 = M[2];
                    const float4 bc = P.mesh_box[2 * mesh], bh = P.mesh_box[2 * mesh + 1];
                    o[0] = m0.x; o[1] = m0.y; o[2] = m0.z; o[3] = m0.w;
                    o[4] = m1.x; o[5] = m1.y; o[6] = m1.z; o[7] = m1.w;
                    o[8] = m2.x; o[9] = m2.y; o[10] = m2.z; o[11] = m2.w;
                    o[12] = bc.x; o[13] = bc.y; o[14] = bc.z;
                    o[15] = bh.x; o[16] = bh.y; o[17] = bh.z;
                }
            }
            __syncwarp();
            if (active && found < 0) {
                for (int k = 0; k < nk; ++k) {
                    const float *o = s_obj[warp][k];
                    if (o[18] == 0.0f) continue;
                    const float d0 = cx - o[3], d1 = cy - o[7], d2 = cz - o[11];
                    float e[3];
#pragma unroll
                    for (int i = 0; i < 3; ++i) {
                        const float loc = fmaf(o[8 + i], d2, fmaf(o[4 + i], d1, o[i] * d0));      // R^T d
                        const float rel = loc - o[12 + i];
                        const float q = fminf(fmaxf(rel, -o[15 + i]), o[15 + i]);
                        e[i] = rel - q;
                    }
                    const float dist2 = fmaf(e[2], e[2], fmaf(e[1], e[1], e[0] * e[0]));
                    if (dist2 <= r2) { found = P.obj_slot0 + k0 + k; break; }
                }
            }
        }
        if (have) {
            P.out_static[(size_t)n * P.S + s] = (uint8_t)hit;
            P.out_object[(size_t)n * P.S + s] = found;
        }
    }
}

}  // namespace gx
