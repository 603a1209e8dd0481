// mdg_camera.cuh — onboard depth / segmentation camera (48 x 64 frames from each
// drone's 60-degree camera at [0.02, 0, 0] in the body frame; "RGB / depth / segmentation cameras").
// The paper renders through OpenGL; this is a ray caster over analytic primitives (readings Q45-Q48): the floor
// plane z = 0 and every other drone of the env as an oblate spheroid.  Product code.
//
// Mapping.  One warp per camera, no block-level synchronisation.  Lanes 0..M-1 prepare one candidate primitive each
// (per-candidate constants of the ray / unit-sphere test in the spheroid's own scaled frame, and a conservative pixel
// bounding box from the bounding sphere); candidates that can be seen are compacted into the warp's shared-memory list.
// Then the 32 lanes sweep the image, four horizontally adjacent pixels per lane and iteration, so a warp stores 512
// contiguous bytes of depth (float4 per lane) and 128 of segmentation (packed u8 x 4 per lane) at a time: the kernel is
// bound by those HBM writes (H W 5 bytes per camera against 32 M bytes of state read).  Spheroids are only intersected
// inside their bounding boxes (see TWO_PASS below), so the common pixel costs the floor test alone.
#pragma once
#include "mdg_dev.cuh"

namespace mdg {

struct CamDev {
    int H, W, groups_per_row, n_groups;     // W / 4, H * W / 4
    int g_rstep, g_cstep;                   // 32 / groups_per_row, 32 % groups_per_row: what a lane's group index advances by per sweep iteration
    float s, half_h, half_w, inv_gpr;       // pixel pitch on the image plane at unit distance; H/2, W/2; 1 / groups_per_row
    float off[3], znear, zfar, rb, inv_a, inv_c;   // rb: radius of the bounding sphere = the larger semi-axis
    float a2, dac;                          // a^2, c^2 - a^2
    float tan_h, tan_v, len_h, len_v;       // W s / 2, H s / 2 and sqrt(1 + tan^2) of each
};

struct __align__(16) CamCand {              // one visible spheroid, in its unit-sphere frame (o = ray origin, d = m0 + y m1 + z m2)
    float w0x, w0y, w0z, w1x, w1y, w1z, w2x, w2y, w2z;   // o x m0, o x m1, o x m2: o x d is linear in (y, z)
    float c00, c01x2, c02x2, c11, c12x2, c22;             // m_a . m_b: |d|^2 is a quadratic in (y, z)
    float b0, b1, b2;                                     // o . m_a
    int id_rpi; float inv_bw;                             // segmentation id | rows per warp pass << 8 (0: box wider than a warp); 1 / box width
    int4 box;                                             // inclusive pixel bounding box (r0, r1, c0, c1)
};

static constexpr int CAM_WARPS = 4;         // cameras per block
// A pixel belongs to a silhouette box when its CENTRE lies within the silhouette's extent widened by this many pixels.  The
// extent comes from the projected conic in fp32 and is good to ~1e-3 pixel (its error scales with the silhouette's size); a
// centre that close to the outline is a tie for the ray test anyway.
static constexpr float CAM_BOX_SLACK = 0.05f;

__device__ __forceinline__ void cam_rotmat(float w, float x, float y, float z, float R[3][3]) {
    R[0][0] = 1.0f - 2.0f * (y * y + z * z); R[0][1] = 2.0f * (x * y - w * z); R[0][2] = 2.0f * (x * z + w * y);
    R[1][0] = 2.0f * (x * y + w * z); R[1][1] = 1.0f - 2.0f * (x * x + z * z); R[1][2] = 2.0f * (y * z - w * x);
    R[2][0] = 2.0f * (x * z - w * y); R[2][1] = 2.0f * (y * z + w * x); R[2][2] = 1.0f - 2.0f * (x * x + y * y);
}

// Ray (1, y, z) of the camera against the unit sphere of candidate q.  The ray misses iff its distance from the centre,
// |o x d| / |d|, exceeds 1; otherwise the front-face parameter is t = -(o.d)/|d|^2 - sqrt((|d|^2 - |o x d|^2)) / |d|^2.
// Both |o x d|^2 and |d|^2 are evaluated from per-candidate constants (9 + 6 words), 14 FMA-class operations per pixel and
// no MUFU on the miss path; every component of o x d is a difference of products formed once per candidate, so the test keeps
// ~1e-5 relative accuracy hundreds of radii away where the textbook discriminant B^2 - A C cancels catastrophically in fp32.
__device__ __forceinline__ bool cam_hit(const CamCand& q, float y, float z, float& t) {
    const float wx = fmaf(y, q.w1x, fmaf(z, q.w2x, q.w0x)), wy = fmaf(y, q.w1y, fmaf(z, q.w2y, q.w0y)), wz = fmaf(y, q.w1z, fmaf(z, q.w2z, q.w0z));
    const float ww = fmaf(wx, wx, fmaf(wy, wy, wz * wz));
    const float A = fmaf(y, fmaf(y, q.c11, fmaf(z, q.c12x2, q.c01x2)), fmaf(z, fmaf(z, q.c22, q.c02x2), q.c00));
    if (ww > A) return false;
    const float rA = rcp_fast(A);
    const float h2 = fmaxf((A - ww) * rA * rA, 1e-30f);
    t = fmaf(-h2, rsqrt_fast(h2), -fmaf(y, q.b1, fmaf(z, q.b2, q.b0)) * rA);
    return true;
}

// TWO_PASS (both outputs requested): the warp first sweeps the floor over the whole image, then visits each candidate's
// bounding box with one lane per PIXEL and depth-tests against what it has just written (still in L2), so no lane idles
// through a spheroid test that cannot concern it.  Otherwise (one output only) a single sweep tests each 4-pixel group
// against the candidates whose box it touches.  Both use cam_hit and the same visiting order (floor, then drones by index;
// strict "<"), so they produce identical images.
// ALIGNED: a row holds a power-of-two number of 4-pixel groups that divides 32 (W = 4 .. 128, the default 64 among them), so a
// lane keeps its columns for the whole sweep and everything that depends on the column only is formed once.
template <bool TWO_PASS, bool ALIGNED>
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
        // bounding sphere against the near / far planes and the four side planes of the view frustum (inward normals
        // (tan, -+1, 0) / sqrt(1 + tan^2) and (tan, 0, -+1) / sqrt(1 + tan^2), tan = half the image extent at unit distance)
        vis = cx + a >= C.znear && cx - a < C.zfar &&
              fmaf(cx, C.tan_h, -fabsf(cy)) >= -a * C.len_h && fmaf(cx, C.tan_v, -fabsf(cz)) >= -a * C.len_v;
        if (vis && cx > 1.1f * a) {
            // Tight box of the silhouette.  In camera coordinates the spheroid's dual quadric projects to the dual conic
            // C* = Sigma - p p^T with Sigma = a^2 I + (c^2 - a^2) n n^T (n = its axis, p = its centre); the image lines u = const
            // (u = Y/X) tangent to the conic solve C*_00 u^2 - 2 C*_01 u + C*_11 = 0, likewise v = Z/X with index 2.  C*_00 < 0
            // because the body lies wholly in front of the plane X = 0 here.  Pixel (r, c) has its centre at (r + 1/2, c + 1/2): the box
            // keeps the pixels whose centre is inside the extent (+- CAM_BOX_SLACK); a silhouette between pixel centres has none.
            const float nx = Ri[0][0] * Rk[0][2] + Ri[1][0] * Rk[1][2] + Ri[2][0] * Rk[2][2];
            const float ny = Ri[0][1] * Rk[0][2] + Ri[1][1] * Rk[1][2] + Ri[2][1] * Rk[2][2];
            const float nz = Ri[0][2] * Rk[0][2] + Ri[1][2] * Rk[1][2] + Ri[2][2] * Rk[2][2];
            const float c00 = fmaf(C.dac, nx * nx, C.a2) - cx * cx;
            const float c01 = C.dac * nx * ny - cx * cy, c11 = fmaf(C.dac, ny * ny, C.a2) - cy * cy;
            const float c02 = C.dac * nx * nz - cx * cz, c22 = fmaf(C.dac, nz * nz, C.a2) - cz * cz;
            const float inv = 1.0f / (c00 * C.s);
            const float su = sqrtf(fmaxf(c01 * c01 - c00 * c11, 0.0f)), sv = sqrtf(fmaxf(c02 * c02 - c00 * c22, 0.0f));
            // column = W/2 - u / s, row = H/2 - v / s; c00 < 0 so (c01 + su) / c00 is the smaller root
            const float ua = (c01 + su) * inv, ub = (c01 - su) * inv, va = (c02 + sv) * inv, vb = (c02 - sv) * inv;
            const float c0 = ceilf(C.half_w - ub - (0.5f + CAM_BOX_SLACK)), c1 = floorf(C.half_w - ua - (0.5f - CAM_BOX_SLACK));
            const float r0 = ceilf(C.half_h - vb - (0.5f + CAM_BOX_SLACK)), r1 = floorf(C.half_h - va - (0.5f - CAM_BOX_SLACK));
            vis = c1 >= c0 && r1 >= r0 && c1 >= 0.0f && c0 <= (float)(C.W - 1) && r1 >= 0.0f && r0 <= (float)(C.H - 1);
            cd.box = make_int4((int)fmaxf(r0, 0.0f), (int)fminf(r1, (float)(C.H - 1)), (int)fmaxf(c0, 0.0f), (int)fminf(c1, (float)(C.W - 1)));
        }
        if (vis) {
            // unit-sphere frame of spheroid k: x' = S R_k^T (x - p_k), S = diag(1/a, 1/a, 1/c)
            const float sc[3] = {C.inv_a, C.inv_a, C.inv_c};
            float o[3], m[3][3];                            // m[c] = image of camera axis c (forward, left, up)
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                o[r] = (Rk[0][r] * rx + Rk[1][r] * ry + Rk[2][r] * rz) * sc[r];
#pragma unroll
                for (int c = 0; c < 3; ++c) m[c][r] = (Rk[0][r] * Ri[0][c] + Rk[1][r] * Ri[1][c] + Rk[2][r] * Ri[2][c]) * sc[r];
            }
            auto crs = [&](const float* v, float& x, float& y, float& z) {
                x = o[1] * v[2] - o[2] * v[1]; y = o[2] * v[0] - o[0] * v[2]; z = o[0] * v[1] - o[1] * v[0];
            };
            auto dot = [](const float* u, const float* v) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; };
            crs(m[0], cd.w0x, cd.w0y, cd.w0z); crs(m[1], cd.w1x, cd.w1y, cd.w1z); crs(m[2], cd.w2x, cd.w2y, cd.w2z);
            cd.c00 = dot(m[0], m[0]); cd.c01x2 = 2.0f * dot(m[0], m[1]); cd.c02x2 = 2.0f * dot(m[0], m[2]);
            cd.c11 = dot(m[1], m[1]); cd.c12x2 = 2.0f * dot(m[1], m[2]); cd.c22 = dot(m[2], m[2]);
            cd.b0 = dot(o, m[0]); cd.b1 = dot(o, m[1]); cd.b2 = dot(o, m[2]);
            const int bw = cd.box.w - cd.box.z + 1;
            cd.id_rpi = (2 + lane) | ((bw <= 32 ? 32 / bw : 0) << 8); cd.inv_bw = 1.0f / (float)bw;
        }
    }
    const unsigned ball = __ballot_sync(0xffffffffu, vis);
    const int n_cand = __popc(ball);
    if (vis) cand[__popc(ball & ((1u << lane) - 1u))] = cd;
    __syncwarp();

    const float noz = oz > 0.0f ? -oz : 0.0f;                    // camera on or under the floor: t = 0 < znear never passes (Q46)
    float* dcam = depth ? depth + (size_t)cam * C.n_groups * 4 : nullptr;
    uint8_t* scam = seg ? seg + (size_t)cam * C.n_groups * 4 : nullptr;
    int r = (int)(((float)lane + 0.5f) * C.inv_gpr), cg = lane - r * C.groups_per_row;   // row and group-in-row of group g
    for (int g = lane; g < C.n_groups; g += 32) {
        const int c4 = cg * 4;
        const float z = (C.half_h - 0.5f - (float)r) * C.s;      // -((r + 1/2) - H/2) s
        const float y0 = (C.half_w - 0.5f - (float)c4) * C.s;
        float y[4], best[4];
        unsigned ids = 0;
        const float dz0 = fmaf(z, Ri[2][2], Ri[2][0]);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            y[j] = fmaf(-(float)j, C.s, y0);
            const float dz = fmaf(y[j], Ri[2][1], dz0);          // world z of the ray direction (1, y, z)
            const float t = noz * rcp_fast(dz);                  // floor: o_z + t d_z = 0; d_z >= 0 gives t <= 0 (or NaN): no hit
            const bool hit = t >= C.znear && t < C.zfar;
            best[j] = hit ? t : C.zfar; ids |= hit ? (1u << (8 * j)) : 0u;
        }
        if (!TWO_PASS) {
            for (int k = 0; k < n_cand; ++k) {
                const CamCand& q = cand[k];
                const int4 bb = q.box;
                if (r < bb.x || r > bb.y || c4 + 3 < bb.z || c4 > bb.w) continue;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    float t;
                    if (cam_hit(q, y[j], z, t) && t >= C.znear && t < best[j]) { best[j] = t; ids = (ids & ~(0xffu << (8 * j))) | ((unsigned)(q.id_rpi & 255) << (8 * j)); }
                }
            }
            if (dcam) __stcs(reinterpret_cast<float4*>(dcam) + g, make_float4(best[0], best[1], best[2], best[3]));
            if (scam) __stcs(reinterpret_cast<unsigned*>(scam) + g, ids);
        } else {
            reinterpret_cast<float4*>(dcam)[g] = make_float4(best[0], best[1], best[2], best[3]);
            reinterpret_cast<unsigned*>(scam)[g] = ids;
        }
        r += C.g_rstep;
        if (!ALIGNED) { cg += C.g_cstep; if (cg >= C.groups_per_row) { cg -= C.groups_per_row; r += 1; } }
    }
    if (TWO_PASS) {
        for (int k = 0; k < n_cand; ++k) {
            __syncwarp();                                        // orders the warp's earlier stores before the loads below
            const CamCand& q = cand[k];
            const int4 bb = q.box;
            const int bw = bb.w - bb.z + 1, rpi = q.id_rpi >> 8;
            const uint8_t id = (uint8_t)(q.id_rpi & 255);
            auto test = [&](int r, int c) {
                const float z = (C.half_h - 0.5f - (float)r) * C.s;
                const float y = fmaf(-(float)(c & 3), C.s, (C.half_w - 0.5f - (float)(c & ~3)) * C.s);   // as the sweep forms it
                float t;
                if (cam_hit(q, y, z, t) && t >= C.znear) {
                    const int px = r * C.W + c;
                    if (t < __ldcg(dcam + px)) { dcam[px] = t; scam[px] = id; }
                }
            };
            if (rpi > 0) {                                       // the usual case: the warp covers rpi whole rows of the box per pass
                const int lr = (int)(((float)lane + 0.5f) * q.inv_bw), c = bb.z + (lane - lr * bw);   // lane / bw, exact for lane, bw <= 32
                if (lr < rpi)
                    for (int r = bb.x + lr; r <= bb.y; r += rpi) test(r, c);
            } else {
                const int n_px = bw * (bb.y - bb.x + 1);
                for (int i = lane; i < n_px; i += 32) {
                    const int rr = (int)(((float)i + 0.5f) * q.inv_bw);
                    test(bb.x + rr, bb.z + (i - rr * bw));
                }
            }
        }
    }
}

}  // namespace mdg
