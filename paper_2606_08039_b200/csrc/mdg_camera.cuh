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

// What the colour frame needs on top (reading Q53): the ray direction in the candidate's unit-sphere frame, d = m0 + y m1 + z m2,
// and L = S R_k^T l, so that for the hit point u (|u| = 1) the shading is n.l = (u.L) / |S u|, |S u|^2 = 1/a^2 + u_z^2 (1/c^2 - 1/a^2).
struct __align__(16) CamShade { float m0[3], m1[3], m2[3], L[3]; unsigned ovl; float pad[3]; };   // ovl: candidates whose box meets this one's

static constexpr int CAM_WARPS = 4;         // cameras per block
enum { CAM_ONE_PASS = 0, CAM_TWO_PASS = 1, CAM_RGBA = 2 };
// Q53: unit vector towards the light, ambient and diffuse weights, sky colour (R | G << 8 | B << 16 | A << 24) and floor albedo
static constexpr float CAM_LIGHT_X = 0.36f, CAM_LIGHT_Y = 0.48f, CAM_LIGHT_Z = 0.80f;
static constexpr float CAM_AMBIENT = 0.3f, CAM_DIFFUSE = 0.7f, CAM_FLOOR_ALBEDO = 160.0f;
static constexpr unsigned CAM_SKY = 135u | (206u << 8) | (235u << 16) | (255u << 24);
__device__ __forceinline__ unsigned cam_shade_rgba(float ar, float ag, float ab, float ndl) {
    const float sh = fmaf(CAM_DIFFUSE, fmaxf(ndl, 0.0f), CAM_AMBIENT);
    return __float2uint_rd(fmaf(ar, sh, 0.5f)) | (__float2uint_rd(fmaf(ag, sh, 0.5f)) << 8) | (__float2uint_rd(fmaf(ab, sh, 0.5f)) << 16) | (255u << 24);
}
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
// n.l at the front hit of ray (1, y, z) on candidate q (the ray is known to hit).  The hit point in the unit-sphere frame is the
// foot of the perpendicular from the centre, d x (o x d) / |d|^2 (|.| <= 1, formed from the same cancellation-free o x d as the
// hit test), minus the half-chord h d: no difference of the large vectors o and t d is ever taken.
__device__ __forceinline__ float cam_ndotl(const CamCand& q, const CamShade& sh, float y, float z, float ia2, float dic) {
    const float wx = fmaf(y, q.w1x, fmaf(z, q.w2x, q.w0x)), wy = fmaf(y, q.w1y, fmaf(z, q.w2y, q.w0y)), wz = fmaf(y, q.w1z, fmaf(z, q.w2z, q.w0z));
    const float ww = fmaf(wx, wx, fmaf(wy, wy, wz * wz));
    const float A = fmaf(y, fmaf(y, q.c11, fmaf(z, q.c12x2, q.c01x2)), fmaf(z, fmaf(z, q.c22, q.c02x2), q.c00));
    const float rA = rcp_fast(A);
    const float h2 = fmaxf((A - ww) * rA * rA, 1e-30f);
    const float h = h2 * rsqrt_fast(h2);
    const float dx = fmaf(y, sh.m1[0], fmaf(z, sh.m2[0], sh.m0[0])), dy = fmaf(y, sh.m1[1], fmaf(z, sh.m2[1], sh.m0[1])), dz = fmaf(y, sh.m1[2], fmaf(z, sh.m2[2], sh.m0[2]));
    const float ux = fmaf(fmaf(dy, wz, -dz * wy), rA, -h * dx), uy = fmaf(fmaf(dz, wx, -dx * wz), rA, -h * dy), uz = fmaf(fmaf(dx, wy, -dy * wx), rA, -h * dz);
    return fmaf(ux, sh.L[0], fmaf(uy, sh.L[1], uz * sh.L[2])) * rsqrt_fast(fmaf(uz * uz, dic, ia2));
}

// TWO_PASS (both outputs requested): the warp first sweeps the floor over the whole image, then visits each candidate's
// bounding box with one lane per PIXEL and depth-tests against what it has just written (still in L2), so no lane idles
// through a spheroid test that cannot concern it.  Otherwise (one output only) a single sweep tests each 4-pixel group
// against the candidates whose box it touches.  Both use cam_hit and the same visiting order (floor, then drones by index;
// strict "<"), so they produce identical images.
// ALIGNED: a row holds a power-of-two number of 4-pixel groups that divides 32 (W = 4 .. 128, the default 64 among them), so a
// lane keeps its columns for the whole sweep and everything that depends on the column only is formed once.
// The candidates' bounding boxes, one after the other, one lane per box pixel: visit(k, q, row, column, y, z, t) for every pixel
// whose ray (1, y, z) hits candidate k in front of the near plane.  Lanes of one call touch different pixels; calls are ordered by __syncwarp.
template <class F>
__device__ __forceinline__ void cam_box_pass(const CamCand* cand, int n_cand, int lane, const CamDev& C, F&& visit) {
    for (int k = 0; k < n_cand; ++k) {
        __syncwarp();                                            // orders the warp's earlier stores before the loads below
        const CamCand& q = cand[k];
        const int4 bb = q.box;
        const int bw = bb.w - bb.z + 1, rpi = q.id_rpi >> 8;
        auto test = [&](int r, int c) {
            const float z = (C.half_h - 0.5f - (float)r) * C.s;
            const float y = fmaf(-(float)(c & 3), C.s, (C.half_w - 0.5f - (float)(c & ~3)) * C.s);   // as the sweep forms it
            float t;
            if (cam_hit(q, y, z, t) && t >= C.znear) visit(k, q, r, c, y, z, t);
        };
        if (rpi > 0) {                                           // the usual case: the warp covers rpi whole rows of the box per pass
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

// MODE = CAM_RGBA: the colour frame (reading Q53) in two passes without any depth buffer.  The sweep writes sky and floor; the
// box pass then decides every drone pixel in registers - a hit wins its pixel when it is in front of the floor and of the hits of
// the few candidates whose boxes meet this one's (CamShade::ovl; same tests, same boxes and the same order rule as the depth
// kernel: the lower drone index wins a tie) - and the winner alone shades and stores its pixel.  Every pixel's final value is
// written by exactly one lane after the sweep's; nothing is read back.  depth and seg are not written.
template <int MODE, bool ALIGNED>
__global__ void __launch_bounds__(CAM_WARPS * 32)
render_depth_kernel(const float4* __restrict__ P0, const float4* __restrict__ P1, int n_cams, int M, const CamDev C,
                    float* __restrict__ depth, uint8_t* __restrict__ seg, uint4* __restrict__ rgba) {
    constexpr bool TWO_PASS = MODE == CAM_TWO_PASS, RGBA = MODE == CAM_RGBA;
    extern __shared__ __align__(16) unsigned char cam_smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int cam = blockIdx.x * CAM_WARPS + wib;
    if (cam >= n_cams) return;
    CamCand* cand = reinterpret_cast<CamCand*>(cam_smem) + (size_t)wib * M;
    CamShade* shade = reinterpret_cast<CamShade*>(cam_smem + (size_t)CAM_WARPS * M * sizeof(CamCand)) + (size_t)wib * M;   // CAM_RGBA only
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
    CamShade sd;
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
            if (RGBA) {
#pragma unroll
                for (int r = 0; r < 3; ++r) {
                    sd.m0[r] = m[0][r]; sd.m1[r] = m[1][r]; sd.m2[r] = m[2][r];
                    sd.L[r] = (Rk[0][r] * CAM_LIGHT_X + Rk[1][r] * CAM_LIGHT_Y + Rk[2][r] * CAM_LIGHT_Z) * sc[r];
                }
            }
            const int bw = cd.box.w - cd.box.z + 1;
            cd.id_rpi = (2 + lane) | ((bw <= 32 ? 32 / bw : 0) << 8); cd.inv_bw = 1.0f / (float)bw;
        }
    }
    const unsigned ball = __ballot_sync(0xffffffffu, vis);
    const int n_cand = __popc(ball);
    if (vis) cand[__popc(ball & ((1u << lane) - 1u))] = cd;
    if (RGBA && vis) shade[__popc(ball & ((1u << lane) - 1u))] = sd;
    __syncwarp();

    if (RGBA) {                                                  // which other candidates can cover a pixel of this one's box
        if (lane < n_cand) {
            const int4 b = cand[lane].box;
            unsigned ovl = 0;
            for (int k = 0; k < n_cand; ++k) {
                const int4 o = cand[k].box;
                if (k != lane && o.x <= b.y && o.y >= b.x && o.z <= b.w && o.w >= b.z) ovl |= 1u << k;
            }
            shade[lane].ovl = ovl;
        }
        __syncwarp();
    }
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
        if (RGBA) {
            const unsigned floor_px = cam_shade_rgba(CAM_FLOOR_ALBEDO, CAM_FLOOR_ALBEDO, CAM_FLOOR_ALBEDO, CAM_LIGHT_Z);
            rgba[(size_t)cam * C.n_groups + g] = make_uint4((ids & 1u) ? floor_px : CAM_SKY, (ids & 0x100u) ? floor_px : CAM_SKY,
                                                            (ids & 0x10000u) ? floor_px : CAM_SKY, (ids & 0x1000000u) ? floor_px : CAM_SKY);
        } else if (!TWO_PASS) {
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
    if (TWO_PASS)
        cam_box_pass(cand, n_cand, lane, C, [&](int, const CamCand& q, int r, int c, float, float, float t) {
            const int px = r * C.W + c;
            if (t < __ldcg(dcam + px)) { dcam[px] = t; scam[px] = (uint8_t)(q.id_rpi & 255); }
        });
    if (RGBA) {
        unsigned* const frame = reinterpret_cast<unsigned*>(rgba) + (size_t)cam * C.n_groups * 4;
        const float ia2 = C.inv_a * C.inv_a, dic = fmaf(C.inv_c, C.inv_c, -ia2);
        cam_box_pass(cand, n_cand, lane, C, [&](int k, const CamCand& q, int r, int c, float y, float z, float t) {
            const float tf = noz * rcp_fast(fmaf(y, Ri[2][1], fmaf(z, Ri[2][2], Ri[2][0])));     // the floor, as the sweep forms it
            bool win = t < ((tf >= C.znear && tf < C.zfar) ? tf : C.zfar);
            for (unsigned others = shade[k].ovl; others; others &= others - 1u) {
                const int k2 = __ffs((int)others) - 1;
                const CamCand& q2 = cand[k2];
                const int4 bb = q2.box;
                float t2;
                if (r >= bb.x && r <= bb.y && c >= bb.z && c <= bb.w && cam_hit(q2, y, z, t2) && t2 >= C.znear && (t2 < t || (t2 == t && k2 < k))) win = false;
            }
            if (win) {
                const int kd = (q.id_rpi & 255) - 2;                 // drone index -> albedo (Q53)
                frame[r * C.W + c] = cam_shade_rgba((float)(250 - 22 * (kd & 7)), (float)(60 + 40 * ((kd >> 3) & 3)), (float)(40 + 26 * (kd & 7)),
                                                    cam_ndotl(q, shade[k], y, z, ia2, dic));
            }
        });
    }
}

}  // namespace mdg
