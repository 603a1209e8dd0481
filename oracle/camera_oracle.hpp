// oracle/camera_oracle.hpp — TEST INFRASTRUCTURE: the plain float64 CPU oracle of the onboard depth /
// segmentation camera ("(N, 48, 64, 4) uint8 frames from each drone's
// onboard 60°-FOV camera, positioned at [0.02, 0, 0] in the body frame"; "RGB / depth /
// segmentation cameras").
//
// The paper renders through mujoco.Renderer (OpenGL): unavailable on this box.  What is built instead is
// a ray caster over analytic primitives, and this file is its definition written out: one ray per pixel,
// every primitive intersected by its textbook quadratic / linear equation, the nearest admissible hit wins.
// Scalar loops camera -> row -> column -> primitive; no culling, no blocking, no reuse between pixels.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may use it; it shares nothing with
// the CUDA path.  Readings (DESIGN.md §3 Q45-Q48):
//   Q45 camera: origin p + R(q) offset; optical axis body +x, image right = body -y, image up = body +z;
//       60° is the VERTICAL field of view (MuJoCo's fovy); H rows x W columns, square pixels, pixel (r, c) looks
//       along the body-frame direction (1, -(c + 1/2 - W/2) s, -(r + 1/2 - H/2) s), s = 2 tan(fovy/2) / H
//       (row 0 = top, column 0 = left).
//   Q46 scene: the floor plane z = 0 seen from above (camera origin z > 0 and ray pointing down), and every
//       OTHER drone of the same env as an oblate spheroid centred on its position, oriented by its quaternion,
//       semi-axes (a, a, c) in its body frame (a = arm + propeller radius, c = half the airframe height);
//       only the front face (near root) of a spheroid is visible; the own airframe is not drawn.
//   Q47 depth = distance along the optical axis in metres (the ray parameter t of the direction above, whose
//       axial component is 1), hits with t < znear or t >= zfar are discarded, background depth = zfar.
//   Q48 segmentation id (u8): 0 background, 1 floor, 2 + k drone k of the env.
//   Q53 colour frame ("(N, 48, 64, 4) uint8"): flat Lambert shading of the same nearest hit.  One directional
//       light, the unit vector towards it l = (0.36, 0.48, 0.80) in the world frame; shade = 0.3 + 0.7 max(0, n.l) with n the
//       outward unit normal of the primitive at the hit point (floor: +z; spheroid: the normalised gradient of its quadric);
//       albedo (R, G, B) in 0..255: floor (160, 160, 160), drone k (250 - 22 (k mod 8), 60 + 40 ((k div 8) mod 4),
//       40 + 26 (k mod 8)) - all even, so that the ambient term alone (0.3 x albedo) never lands on a rounding boundary; channel = floor(albedo * shade + 1/2); background = the unshaded sky (135, 206, 235); alpha = 255.
// Pins (tests/test_oracle_camera.py): floor depth rows of a level camera against the similar-triangles value
// h / tan(elevation); forward pinhole projection of small spheres at tabulated bearings lands in the pixel the
// ray caster marks (tests/golden/camera_bearings.txt); on-axis sphere silhouette area and nearest depth d - R;
// every hit pixel's reconstructed 3-D point lies on its primitive; yaw co-rotation invariance; roll by pi flips
// the image; occlusion order; a : c aspect of a spheroid seen edge-on; spheroid seen along its axis = disc of radius a.
// Colour frame (tests/test_oracle_camera_rgba.py): the floor's hand value; a sphere's radial normals; the finite-difference
// gradient of the defining quadric for tilted spheroids; back-lit faces = the ambient term alone; sky and alpha.
#pragma once
#include <cmath>
#include <cstdint>

#include "drone_oracle.hpp"

namespace orc {

struct CamParams {
    int H, W;
    double fovy_deg, offset[3], znear, zfar, body_a, body_c;
};

// One camera image.  state: [n_drones][13] = p(3) q(4: w x y z) v(3) w(3) of the env's drones; i = the drone that
// carries the camera.  depth / seg: [H*W]; margin (may be null): per pixel, the smallest relative distance of any
// decision taken for it (discriminant sign, near / far clip, ordering of the two nearest hits, floor side) to its
// threshold, so that a comparison in another precision can tell a tie from an error.
// rgba (may be null): [H*W][4] u8 of reading Q53; shade_out (may be null): per pixel, the shade before quantisation (1 for the
// background), so that a comparison in another precision can tell a value next to a rounding boundary from an error.
constexpr double LIGHT_DIR[3] = {0.36, 0.48, 0.80};
constexpr double SHADE_AMBIENT = 0.3, SHADE_DIFFUSE = 0.7;
inline void albedo_of(int id, double rgb[3]) {
    if (id == 0) { rgb[0] = 135.0; rgb[1] = 206.0; rgb[2] = 235.0; }
    else if (id == 1) { rgb[0] = rgb[1] = rgb[2] = 160.0; }
    else {
        const int k = id - 2;
        rgb[0] = 250.0 - 22.0 * (k % 8); rgb[1] = 60.0 + 40.0 * ((k / 8) % 4); rgb[2] = 40.0 + 26.0 * (k % 8);
    }
}

inline void render_camera(const double* state, int n_drones, int i, const CamParams& cp, double* depth, uint8_t* seg,
                          double* margin, uint8_t* rgba = nullptr, double* shade_out = nullptr) {
    const double* si = state + 13 * i;
    double Ri[3][3], o[3], off_w[3];
    rotmat(si + 3, Ri);
    mat_vec(Ri, cp.offset, off_w);
    for (int a = 0; a < 3; ++a) o[a] = si[a] + off_w[a];
    const double s = 2.0 * std::tan(0.5 * cp.fovy_deg * PI / 180.0) / cp.H;
    for (int r = 0; r < cp.H; ++r) {
        for (int c = 0; c < cp.W; ++c) {
            const double d_b[3] = {1.0, -((c + 0.5) - 0.5 * cp.W) * s, -((r + 0.5) - 0.5 * cp.H) * s};
            double d[3];
            mat_vec(Ri, d_b, d);
            double best = cp.zfar, second = INFINITY, mg = INFINITY;
            int id = 0;
            auto consider = [&](double t, int ident) {     // Q47: admissible range, nearest wins
                mg = std::fmin(mg, std::fabs(t - cp.znear) / cp.znear);
                mg = std::fmin(mg, std::fabs(t - cp.zfar) / cp.zfar);
                if (t < cp.znear || t >= cp.zfar) return;
                if (t < best) { second = best; best = t; id = ident; }
                else if (t < second) second = t;
            };
            // floor (Q46)
            mg = std::fmin(mg, std::fabs(o[2]) / 1e-3);
            if (o[2] > 0.0 && d[2] < 0.0) consider(-o[2] / d[2], 1);
            // the other drones of the env (Q46): |S^-1 R_k^T (o + t d - p_k)|^2 = 1
            for (int k = 0; k < n_drones; ++k) {
                if (k == i) continue;
                const double* sk = state + 13 * k;
                double Rk[3][3], rel[3], ob[3], db[3];
                rotmat(sk + 3, Rk);
                for (int a = 0; a < 3; ++a) rel[a] = o[a] - sk[a];
                matT_vec(Rk, rel, ob);
                matT_vec(Rk, d, db);
                const double inv[3] = {1.0 / cp.body_a, 1.0 / cp.body_a, 1.0 / cp.body_c};
                double A = 0.0, B = 0.0, Cc = -1.0;
                for (int a = 0; a < 3; ++a) {
                    const double os = ob[a] * inv[a], ds = db[a] * inv[a];
                    A += ds * ds; B += os * ds; Cc += os * os;
                }
                const double disc = B * B - A * Cc;
                mg = std::fmin(mg, std::fabs(disc) / A);       // = |1 - (miss distance / radius)^2| in the unit-sphere frame
                if (disc < 0.0) continue;
                consider((-B - std::sqrt(disc)) / A, 2 + k);
            }
            if (id != 0 && std::isfinite(second)) mg = std::fmin(mg, (second - best) / best);
            depth[r * cp.W + c] = best;
            seg[r * cp.W + c] = (uint8_t)id;
            if (margin) margin[r * cp.W + c] = mg;
            if (rgba) {                                        // Q53
                double shade = 1.0, alb[3];
                albedo_of(id, alb);
                if (id != 0) {
                    double n[3] = {0.0, 0.0, 1.0};
                    if (id >= 2) {
                        const double* sk = state + 13 * (id - 2);
                        double Rk[3][3], rel[3], b[3], g[3];
                        rotmat(sk + 3, Rk);
                        for (int a = 0; a < 3; ++a) rel[a] = o[a] + best * d[a] - sk[a];      // hit point relative to the body's centre
                        matT_vec(Rk, rel, b);
                        const double ia2 = 1.0 / (cp.body_a * cp.body_a), ic2 = 1.0 / (cp.body_c * cp.body_c);
                        const double gb[3] = {b[0] * ia2, b[1] * ia2, b[2] * ic2};              // gradient of x^2/a^2 + y^2/a^2 + z^2/c^2 (halved)
                        mat_vec(Rk, gb, g);
                        const double gn = std::sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
                        for (int a = 0; a < 3; ++a) n[a] = g[a] / gn;
                    }
                    const double ndl = n[0] * LIGHT_DIR[0] + n[1] * LIGHT_DIR[1] + n[2] * LIGHT_DIR[2];
                    shade = SHADE_AMBIENT + SHADE_DIFFUSE * std::fmax(0.0, ndl);
                }
                for (int ch = 0; ch < 3; ++ch) rgba[(r * cp.W + c) * 4 + ch] = (uint8_t)std::floor(alb[ch] * shade + 0.5);
                rgba[(r * cp.W + c) * 4 + 3] = 255;
                if (shade_out) shade_out[r * cp.W + c] = shade;
            }
        }
    }
}

}  // namespace orc
