// mdg_camera.cuh — onboard depth / segmentation camera (48 x 64 frames from each
// drone's 60-degree camera at [0.02, 0, 0] in the body frame; "RGB / depth / segmentation cameras").
// The paper renders through OpenGL; this is a ray caster over analytic primitives (readings Q45-Q48): the floor
// plane z = 0 and every other drone of the env as an oblate spheroid.  Product code.
//
// Mapping.  One warp per camera, no block-level synchronisation.  Lanes 0..M-1 prepare one candidate primitive each
// (the ray origin and the three columns of S R_k^T R_i in the spheroid's unit-sphere frame, and a conservative pixel
// bounding box from the bounding sphere); candidates that can be seen are compacted into the warp's shared-memory list.
// Then the 32 lanes sweep the image, four horizontally adjacent pixels per lane and iteration, so a warp stores 512
// contiguous bytes of depth (float4 per lane) and 128 of segmentation (uchar4 per lane) at a time: the kernel is bound
// by those HBM writes (H W 5 bytes per camera against 32 M bytes of state read).  A spheroid is only intersected for
// pixel groups inside its bounding box, so the common pixel costs the floor test alone.
//
// Arithmetic.  The quadratic is solved around the point of closest approach (t_c = -B/A, v = o + t_c d, hit iff |v| < 1,
// t = t_c - sqrt((1 - |v|^2)/A)), which keeps fp32 accurate when the camera is hundreds of radii away (the textbook
// discriminant B^2 - A C cancels catastrophically there).
#pragma once
#include "mdg_dev.cuh"

namespace mdg {

struct CamDev {
    int H, W, groups_per_row, n_groups;     // W / 4, H * W / 4
    float s, half_h, half_w, inv_gpr;       // pixel pitch on the image plane at unit distance; H/2, W/2; 1 / groups_per_row
    float off[3], znear, zfar, rb, inv_a, inv_c;   // rb: radius of the bounding sphere = the larger semi-axis
};

struct __align__(16) CamCand {                            // one visible spheroid, in its unit-sphere frame
    float ox, oy, oz;                       // ray origin
    float m0x, m0y, m0z, m1x, m1y, m1z, m2x, m2y, m2z;   // image of the camera axes (forward, pixel-right * -1, pixel-up): d = m0 + y m1 + z m2
    int4 box; int id;                       // inclusive pixel bounding box (r0, r1, c0, c1), segmentation id
};

static constexpr int CAM_WARPS = 4;         // cameras per block

__device__ __forceinline__ void cam_rotmat(float w, float x, float y, float z, float R[3][3]) {
    R[0][0] = 1.0f - 2.0f * (y * y + z * z); R[0][1] = 2.0f * (x * y - w * z); R[0][2] = 2.0f * (x * z + w * y);
    R[1][0] = 2.0f * (x * y + w * z); R[1][1] = 1.0f - 2.0f * (x * x + z * z); R[1][2] = 2.0f * (y * z - w * x);
    R[2][0] = 2.0f * (x * z - w * y); R[2][1] = 2.0f * (y * z + w * x); R[2][2] = 1.0f - 2.0f * (x * x + y * y);
}

__global__ void __launch_bounds__(CAM_WARPS * 32)
render_depth_kernel(const float4* __restrict__ P0, const float4* __restrict__ P1, int n_cams, int M, const CamDev C,
                    float* __restrict__ depth, uint8_t* __restrict__ seg) {
    extern __shared__ __align__(16) unsigned char cam_smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int cam = blockIdx.x * CAM_WARPS + wib;
    if (cam >= n_cams) return;
    CamCand* cand = reinterpret_cast<CamCand*>(cam_smem) + (size_t)wib * M;
    const int env0 = (cam / M) * M, self = cam - env0;

    // camera pose (every lane; the loads are warp-uniform broadcasts)
    const float4 a0 = __ldg(P0 + cam), a1 = __ldg(P1 + cam);
    float Ri[3][3];
    cam_rotmat(a0.w, a1.x, a1.y, a1.z, Ri);
    const float ox = a0.x + (Ri[0][0] * C.off[0] + Ri[0][1] * C.off[1] + Ri[0][2] * C.off[2]);
    const float oy = a0.y + (Ri[1][0] * C.off[0] + Ri[1][1] * C.off[1] + Ri[1][2] * C.off[2]);
    const float oz = a0.z + (Ri[2][0] * C.off[0] + Ri[2][1] * C.off[1] + Ri[2][2] * C.off[2]);

    // candidate list: lane k prepares drone k of the env
    bool vis = false;
    CamCand cd;
    if (lane < M && lane != self) {
        const float4 b0 = __ldg(P0 + env0 + lane), b1 = __ldg(P1 + env0 + lane);
        float Rk[3][3];
        cam_rotmat(b0.w, b1.x, b1.y, b1.z, Rk);
        const float rx = ox - b0.x, ry = oy - b0.y, rz = oz - b0.z;
        // bounding sphere of radius a, centre in the camera frame (x forward, y left, z up)
        const float cx = -(Ri[0][0] * rx + Ri[1][0] * ry + Ri[2][0] * rz);
        const float cy = -(Ri[0][1] * rx + Ri[1][1] * ry + Ri[2][1] * rz);
        const float cz = -(Ri[0][2] * rx + Ri[1][2] * ry + Ri[2][2] * rz);
        const float a = C.rb * 1.001f;
        cd.box = make_int4(0, C.H - 1, 0, C.W - 1);
        vis = cx + a >= C.znear && cx - a < C.zfar;
        if (vis && cx > 1.5f * a) {
            // a point c + a n of the sphere projects to y/x with |y/x - cy/cx| <= a sqrt(cx^2 + cy^2) / (cx (cx - a))
            const float inv = 1.0f / (cx * (cx - a) * C.s);
            const float du = a * sqrtf(cx * cx + cy * cy) * inv + 1.0f, dv = a * sqrtf(cx * cx + cz * cz) * inv + 1.0f;
            const float uc = C.half_w - cy / (cx * C.s), vc = C.half_h - cz / (cx * C.s);     // column, row of the centre
            const float c0 = floorf(uc - du), c1 = ceilf(uc + du), r0 = floorf(vc - dv), r1 = ceilf(vc + dv);
            vis = c1 >= 0.0f && c0 <= (float)(C.W - 1) && r1 >= 0.0f && r0 <= (float)(C.H - 1);
            cd.box = make_int4((int)fmaxf(r0, 0.0f), (int)fminf(r1, (float)(C.H - 1)), (int)fmaxf(c0, 0.0f), (int)fminf(c1, (float)(C.W - 1)));
        }
        if (vis) {
            // unit-sphere frame of spheroid k: x' = S R_k^T (x - p_k), S = diag(1/a, 1/a, 1/c)
            const float sc[3] = {C.inv_a, C.inv_a, C.inv_c};
            float o[3], m[3][3];
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                o[r] = (Rk[0][r] * rx + Rk[1][r] * ry + Rk[2][r] * rz) * sc[r];
#pragma unroll
                for (int c = 0; c < 3; ++c) m[c][r] = (Rk[0][r] * Ri[0][c] + Rk[1][r] * Ri[1][c] + Rk[2][r] * Ri[2][c]) * sc[r];
            }
            cd.ox = o[0]; cd.oy = o[1]; cd.oz = o[2];
            cd.m0x = m[0][0]; cd.m0y = m[0][1]; cd.m0z = m[0][2];
            cd.m1x = m[1][0]; cd.m1y = m[1][1]; cd.m1z = m[1][2];
            cd.m2x = m[2][0]; cd.m2y = m[2][1]; cd.m2z = m[2][2];
            cd.id = 2 + lane;
        }
    }
    const unsigned ball = __ballot_sync(0xffffffffu, vis);
    const int n_cand = __popc(ball);
    if (vis) cand[__popc(ball & ((1u << lane) - 1u))] = cd;
    __syncwarp();

    const float noz = oz > 0.0f ? -oz : 0.0f;                    // camera on or under the floor: t = 0 < znear never passes (Q46)
    float* dcam = depth ? depth + (size_t)cam * C.n_groups * 4 : nullptr;
    uint8_t* scam = seg ? seg + (size_t)cam * C.n_groups * 4 : nullptr;
    for (int g = lane; g < C.n_groups; g += 32) {
        const int r = (int)(((float)g + 0.5f) * C.inv_gpr);      // exact for g < 2^22
        const int c4 = (g - r * C.groups_per_row) * 4;
        const float z = (C.half_h - 0.5f - (float)r) * C.s;      // -((r + 1/2) - H/2) s
        const float y0 = (C.half_w - 0.5f - (float)c4) * C.s;
        float y[4], best[4];
        int id[4];
        const float dz0 = fmaf(z, Ri[2][2], Ri[2][0]);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            y[j] = fmaf(-(float)j, C.s, y0);
            const float dz = fmaf(y[j], Ri[2][1], dz0);          // world z of the ray direction (1, y, z)
            const float t = noz * rcp_fast(dz);                  // floor: o_z + t d_z = 0
            const bool hit = dz < 0.0f && t >= C.znear && t < C.zfar;
            best[j] = hit ? t : C.zfar; id[j] = hit ? 1 : 0;
        }
        for (int k = 0; k < n_cand; ++k) {
            const CamCand& q = cand[k];
            const int4 bb = q.box;                               // r0, r1, c0, c1
            if (r < bb.x || r > bb.y || c4 + 3 < bb.z || c4 > bb.w) continue;
            const float bx = fmaf(z, q.m2x, q.m0x), by = fmaf(z, q.m2y, q.m0y), bz = fmaf(z, q.m2z, q.m0z);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float dx = fmaf(y[j], q.m1x, bx), dy = fmaf(y[j], q.m1y, by), dzz = fmaf(y[j], q.m1z, bz);
                const float A = fmaf(dx, dx, fmaf(dy, dy, dzz * dzz));
                const float Bq = fmaf(q.ox, dx, fmaf(q.oy, dy, q.oz * dzz));
                const float rA = rcp_fast(A);
                const float tc = -Bq * rA;
                const float vx = fmaf(tc, dx, q.ox), vy = fmaf(tc, dy, q.oy), vz = fmaf(tc, dzz, q.oz);
                const float vv = fmaf(vx, vx, fmaf(vy, vy, vz * vz));
                if (vv <= 1.0f) {
                    const float h2 = fmaxf((1.0f - vv) * rA, 1e-30f);
                    const float t = fmaf(-h2, rsqrt_fast(h2), tc);
                    if (t >= C.znear && t < best[j]) { best[j] = t; id[j] = q.id; }
                }
            }
        }
        if (dcam) __stcs(reinterpret_cast<float4*>(dcam) + g, make_float4(best[0], best[1], best[2], best[3]));
        if (scam) __stcs(reinterpret_cast<unsigned*>(scam) + g, (unsigned)id[0] | ((unsigned)id[1] << 8) | ((unsigned)id[2] << 16) | ((unsigned)id[3] << 24));
    }
}

}  // namespace mdg
