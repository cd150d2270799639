// gx_fk.cuh -- the scene-graph update of gx_update_transforms (sm_100a): forward kinematics from base pose and
// joint positions to the link, camera and held-object transforms gx_render_batch reads (N12;
// PAPER.md:91, 109; it replaces the CPU "Render Setup" stage of Table 5).
// Arithmetic follows N12 operation by operation (compiled with -fmad=false: only the fmaf() calls fuse).
// Product code: nothing here is shared with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace gx {

constexpr int FK_MAX_LINKS = 64;

struct FkLink {          // device copy of a GxLink
    int32_t parent, joint_type;
    float axis[3];
    float origin[12];
};

struct FkParams {
    const FkLink *links;
    int32_t L, camera_link, ee_link;
    float cam_mount[12];
    int32_t N, K, link_slot0;
    const float *base_pose;      // [N,3] x, z, yaw
    const float *joint_pos;      // [N,L]
    const int32_t *held_slot;    // [N] or NULL
    const float *held_xform;     // [N,12] or NULL
    float *cam_pose;             // [N,16]
    float *inst_xform;           // [N,K,16]
};

// N12a: binary32 sine and cosine (Cody-Waite reduction by pi/2 in two steps, minimax polynomials, quadrant)
__device__ __forceinline__ void fk_sincos(float x, float &s, float &c) {
    const float k = rintf(x * 0.636619772f);
    float r = fmaf(-k, 1.57079625f, x);
    r = fmaf(-k, 7.54978942e-08f, r);
    const float z = r * r;
    float ps = fmaf(z, -1.9515295891e-4f, 8.3321608736e-3f);
    ps = fmaf(z, ps, -1.6666654611e-1f);
    const float sn = fmaf(r * z, ps, r);
    float pc = fmaf(z, 2.443315711809948e-5f, -1.388731625493765e-3f);
    pc = fmaf(z, pc, 4.166664568298827e-2f);
    const float cs = fmaf(z * z, pc, fmaf(-0.5f, z, 1.0f));
    const int q = (int)k & 3;
    s = (q & 1) ? cs : sn;
    c = (q & 1) ? sn : cs;
    if (q == 1 || q == 2) c = -c;
    if (q >= 2) s = -s;
}

// C = A * B, 3x4 affine, the operation order of N2
__device__ __forceinline__ void fk_mul(const float *A, const float *B, float *C) {
#pragma unroll
    for (int i = 0; i < 3; ++i) {
#pragma unroll
        for (int j = 0; j < 3; ++j)
            C[i * 4 + j] = fmaf(A[i * 4 + 2], B[8 + j], fmaf(A[i * 4 + 1], B[4 + j], A[i * 4] * B[j]));
        C[i * 4 + 3] = fmaf(A[i * 4 + 2], B[11], fmaf(A[i * 4 + 1], B[7], fmaf(A[i * 4], B[3], A[i * 4 + 3])));
    }
}

__device__ __forceinline__ void fk_store44(float *dst, const float *M) {
    float4 *d = reinterpret_cast<float4 *>(dst);   // (16-float rows of a cudaMalloc'ed array: 16-byte aligned)
    d[0] = make_float4(M[0], M[1], M[2], M[3]);
    d[1] = make_float4(M[4], M[5], M[6], M[7]);
    d[2] = make_float4(M[8], M[9], M[10], M[11]);
    d[3] = make_float4(0.0f, 0.0f, 0.0f, 1.0f);
}

// One warp per environment.  Step 1, lane l < L: the local transform O_l * J_l(theta) of link l (the sine / cosine
// and the Rodrigues matrix, the expensive part, in parallel over the links) into shared memory.  Step 2, lane 0
// walks the chain W_l = W_parent * local_l (a parent precedes its children) and leaves every W_l in shared memory.
// Step 3, the lanes store the link transforms, the camera pose and the held object's transform.
template <int WARPS>
__global__ void __launch_bounds__(WARPS * 32) fk_kernel(const FkParams P) {
    __shared__ float s_loc[WARPS][FK_MAX_LINKS + 1][12];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = blockIdx.x * WARPS + warp;
    if (n >= P.N) return;
    float(*W)[12] = s_loc[warp];      // W[0] = base, W[l + 1] = link l (first its local transform, then its world one)
    const int L = P.L;
    for (int l = lane; l < L; l += 32) {
        const FkLink lk = P.links[l];
        const float th = P.joint_pos[(size_t)n * L + l];
        float J[12];
#pragma unroll
        for (int k = 0; k < 12; ++k) J[k] = (k % 5 == 0) ? 1.0f : 0.0f;
        if (lk.joint_type == 1) {
            float s, c;
            fk_sincos(th, s, c);
            const float t = 1.0f - c;
            const float a0 = lk.axis[0], a1 = lk.axis[1], a2 = lk.axis[2];
            J[0] = fmaf(t * a0, a0, c);
            J[1] = fmaf(t * a0, a1, -(s * a2));
            J[2] = fmaf(t * a0, a2, s * a1);
            J[4] = fmaf(t * a1, a0, s * a2);
            J[5] = fmaf(t * a1, a1, c);
            J[6] = fmaf(t * a1, a2, -(s * a0));
            J[8] = fmaf(t * a2, a0, -(s * a1));
            J[9] = fmaf(t * a2, a1, s * a0);
            J[10] = fmaf(t * a2, a2, c);
        } else if (lk.joint_type == 2) {
            J[3] = th * lk.axis[0];
            J[7] = th * lk.axis[1];
            J[11] = th * lk.axis[2];
        }
        float Loc[12];
        fk_mul(lk.origin, J, Loc);
#pragma unroll
        for (int k = 0; k < 12; ++k) W[l + 1][k] = Loc[k];
    }
    if (lane == 0) {
        float s, c;
        fk_sincos(P.base_pose[3 * (size_t)n + 2], s, c);
        const float B[12] = {c, 0.0f, s, P.base_pose[3 * (size_t)n], 0.0f, 1.0f, 0.0f, 0.0f, -s, 0.0f, c, P.base_pose[3 * (size_t)n + 1]};
#pragma unroll
        for (int k = 0; k < 12; ++k) W[0][k] = B[k];
    }
    __syncwarp();
    if (lane == 0) {
        for (int l = 0; l < L; ++l) {
            float Wl[12];
            fk_mul(W[P.links[l].parent + 1], W[l + 1], Wl);
#pragma unroll
            for (int k = 0; k < 12; ++k) W[l + 1][k] = Wl[k];
        }
    }
    __syncwarp();
    for (int l = lane; l < L; l += 32) fk_store44(P.inst_xform + ((size_t)n * P.K + P.link_slot0 + l) * 16, W[l + 1]);
    if (lane == 31) {
        float Cm[12];
        fk_mul(W[P.camera_link + 1], P.cam_mount, Cm);
        fk_store44(P.cam_pose + (size_t)n * 16, Cm);
    }
    if (lane == 30 && P.held_slot && P.held_xform) {
        const int hs = P.held_slot[n];
        if (hs >= 0 && hs < P.K) {
            float H[12], Hm[12];
#pragma unroll
            for (int k = 0; k < 12; ++k) H[k] = P.held_xform[(size_t)n * 12 + k];
            fk_mul(W[P.ee_link + 1], H, Hm);
            fk_store44(P.inst_xform + ((size_t)n * P.K + hs) * 16, Hm);
        }
    }
}

}  // namespace gx
