// gs_oracle.cpp -- CPU ORACLE for the differentiable 3D Gaussian splatting hot path.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
// code, header, table or helper with the CUDA path under paper_2606_11390_b200/csrc/.
//
// What it is: a plain, single-threaded, obviously-correct restatement of the operators the
// paper distributes (§4: "Gaussian spherical harmonics [10] and Gaussian
// projection operators", per-camera depth sort, "Gaussian rasterization"; PAPER.md:98:
// backward with accumulated per-Gaussian gradients).  The paper states no formula and
// defers to its reference [10]; the mathematics followed here is the
// step-by-step definition written out in SURVEY.md §8(c) (O-P1, O-B, O-R1, O-R2, O-P5),
// with the readings A1..A18 listed there and repeated in DESIGN.md.
//
// Every function is a template on Real (double = truth and finite differences,
// float = fp32 noise floor and the timed CPU baseline).  No blocking, fusion or reordering
// beyond what the definition states.  Compile with -ffp-contract=off.
//
// Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): closed-form single isotropic
// Gaussian, SH basis vs a library spherical-harmonic routine and orthonormality by
// quadrature, covariance vs a library rotation, EWA vs numerical Jacobian and Monte-Carlo,
// radius vs a library eigen-solver, brute-force binning, compositing invariants and the
// "over" operator, untiled brute-force rendering, central finite differences for R2/P5.
// Paper-printed worked values: none exist (parity on paper-printed numbers is unpinned).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

// ---------------------------------------------------------------------------------------
// configuration and camera (passed as flat double arrays so that no struct layout is
// shared with the CUDA library)
// cfg[7]  = dilation, alpha_min, alpha_max, t_min, extent, tile, sh_degree
// cam[20] = width, height, fx, fy, cx, cy, near, far, viewmat[12] (row-major 3x4 [W|tau])
// ---------------------------------------------------------------------------------------
struct Cfg {
    double dilation, alpha_min, alpha_max, t_min, extent;
    int tile, deg;
};
Cfg load_cfg(const double* c) {
    Cfg k;
    k.dilation = c[0]; k.alpha_min = c[1]; k.alpha_max = c[2]; k.t_min = c[3]; k.extent = c[4];
    k.tile = (int)c[5]; k.deg = (int)c[6];
    return k;
}
template <class R>
struct Cam {
    int width, height;
    R fx, fy, cx, cy, near_plane, far_plane;
    R W[3][3];
    R tau[3];
};
template <class R>
Cam<R> load_cam(const double* c) {
    Cam<R> k;
    k.width = (int)c[0]; k.height = (int)c[1];
    k.fx = (R)c[2]; k.fy = (R)c[3]; k.cx = (R)c[4]; k.cy = (R)c[5];
    k.near_plane = (R)c[6]; k.far_plane = (R)c[7];
    for (int r = 0; r < 3; ++r) {
        for (int j = 0; j < 3; ++j) k.W[r][j] = (R)c[8 + 4 * r + j];
        k.tau[r] = (R)c[8 + 4 * r + 3];
    }
    return k;
}

// ---------------------------------------------------------------------------------------
// Real spherical-harmonic basis, SURVEY.md §8(c) O-P1 step 9 (closed-form constants).
// ---------------------------------------------------------------------------------------
const double kPi = 3.14159265358979323846;
template <class R>
void sh_basis(R x, R y, R z, R Y[16]) {
    const R c0 = (R)(0.5 / std::sqrt(kPi));
    const R c1 = (R)std::sqrt(3.0 / (4.0 * kPi));
    const R c2a = (R)(0.5 * std::sqrt(15.0 / kPi));
    const R c2b = (R)(0.25 * std::sqrt(5.0 / kPi));
    const R c2c = (R)(0.25 * std::sqrt(15.0 / kPi));
    const R c3a = (R)(0.25 * std::sqrt(35.0 / (2.0 * kPi)));
    const R c3b = (R)(0.5 * std::sqrt(105.0 / kPi));
    const R c3c = (R)(0.25 * std::sqrt(21.0 / (2.0 * kPi)));
    const R c3d = (R)(0.25 * std::sqrt(7.0 / kPi));
    const R c3e = (R)(0.25 * std::sqrt(105.0 / kPi));
    Y[0] = c0;
    Y[1] = -c1 * y;
    Y[2] = c1 * z;
    Y[3] = -c1 * x;
    Y[4] = c2a * x * y;
    Y[5] = -c2a * y * z;
    Y[6] = c2b * (2 * z * z - x * x - y * y);
    Y[7] = -c2a * x * z;
    Y[8] = c2c * (x * x - y * y);
    Y[9] = -c3a * y * (3 * x * x - y * y);
    Y[10] = c3b * x * y * z;
    Y[11] = -c3c * y * (4 * z * z - x * x - y * y);
    Y[12] = c3d * z * (2 * z * z - 3 * x * x - 3 * y * y);
    Y[13] = -c3c * x * (4 * z * z - x * x - y * y);
    Y[14] = c3e * z * (x * x - y * y);
    Y[15] = -c3a * x * (x * x - 3 * y * y);
}
// Gradient of each basis polynomial with respect to (x, y, z) (unconstrained); the
// projection onto the unit sphere's tangent space happens where the direction is normalised.
template <class R>
void sh_basis_grad(R x, R y, R z, R dY[16][3]) {
    const R c1 = (R)std::sqrt(3.0 / (4.0 * kPi));
    const R c2a = (R)(0.5 * std::sqrt(15.0 / kPi));
    const R c2b = (R)(0.25 * std::sqrt(5.0 / kPi));
    const R c2c = (R)(0.25 * std::sqrt(15.0 / kPi));
    const R c3a = (R)(0.25 * std::sqrt(35.0 / (2.0 * kPi)));
    const R c3b = (R)(0.5 * std::sqrt(105.0 / kPi));
    const R c3c = (R)(0.25 * std::sqrt(21.0 / (2.0 * kPi)));
    const R c3d = (R)(0.25 * std::sqrt(7.0 / kPi));
    const R c3e = (R)(0.25 * std::sqrt(105.0 / kPi));
    auto set = [&](int k, R a, R b, R c) { dY[k][0] = a; dY[k][1] = b; dY[k][2] = c; };
    set(0, 0, 0, 0);
    set(1, 0, -c1, 0);
    set(2, 0, 0, c1);
    set(3, -c1, 0, 0);
    set(4, c2a * y, c2a * x, 0);
    set(5, 0, -c2a * z, -c2a * y);
    set(6, -2 * c2b * x, -2 * c2b * y, 4 * c2b * z);
    set(7, -c2a * z, 0, -c2a * x);
    set(8, 2 * c2c * x, -2 * c2c * y, 0);
    set(9, -c3a * 6 * x * y, -c3a * (3 * x * x - 3 * y * y), 0);
    set(10, c3b * y * z, c3b * x * z, c3b * x * y);
    set(11, c3c * 2 * x * y, -c3c * (4 * z * z - x * x - 3 * y * y), -c3c * 8 * y * z);
    set(12, -c3d * 6 * x * z, -c3d * 6 * y * z, c3d * (6 * z * z - 3 * x * x - 3 * y * y));
    set(13, -c3c * (4 * z * z - 3 * x * x - y * y), c3c * 2 * x * y, -c3c * 8 * x * z);
    set(14, c3e * 2 * x * z, -c3e * 2 * y * z, c3e * (x * x - y * y));
    set(15, -c3a * (3 * x * x - 3 * y * y), c3a * 6 * x * y, 0);
}

// ---------------------------------------------------------------------------------------
// O-P1 step 2: s = exp(l); q^ = q/|q| with q = (w,x,y,z); R(q^); M = R diag(s); Sigma = M M^T
// ---------------------------------------------------------------------------------------
template <class R>
void quat_to_rot(const R qh[4], R Rm[3][3]) {
    const R w = qh[0], x = qh[1], y = qh[2], z = qh[3];
    Rm[0][0] = 1 - 2 * (y * y + z * z); Rm[0][1] = 2 * (x * y - w * z);     Rm[0][2] = 2 * (x * z + w * y);
    Rm[1][0] = 2 * (x * y + w * z);     Rm[1][1] = 1 - 2 * (x * x + z * z); Rm[1][2] = 2 * (y * z - w * x);
    Rm[2][0] = 2 * (x * z - w * y);     Rm[2][1] = 2 * (y * z + w * x);     Rm[2][2] = 1 - 2 * (x * x + y * y);
}
template <class R>
void cov3d(const R ls[3], const R q[4], R s[3], R qh[4], R Rm[3][3], R Mm[3][3], R Sig[3][3]) {
    for (int k = 0; k < 3; ++k) s[k] = std::exp(ls[k]);
    const R qn = std::sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    for (int k = 0; k < 4; ++k) qh[k] = q[k] / qn;
    quat_to_rot(qh, Rm);
    for (int r = 0; r < 3; ++r)
        for (int k = 0; k < 3; ++k) Mm[r][k] = Rm[r][k] * s[k];
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) {
            R acc = 0;
            for (int k = 0; k < 3; ++k) acc += Mm[r][k] * Mm[c][k];
            Sig[r][c] = acc;
        }
}

// Per-(Gaussian, camera) forward intermediates that the backward pass re-derives.
template <class R>
struct Proj {
    bool visible;
    R t[3];
    R xt, yt;            // clamped x~, y~ of step 3
    bool clamp_x, clamp_y;
    R J[2][3];
    R T[2][3];
    R a, b, c, det;      // dilated 2-D covariance entries and determinant
    R conic[3];
    R u, v;
    R radius_real;
    int radius;
    int x0, x1, y0, y1;
    uint32_t tiles;
};

// O-P1 step 8: tile rectangle, evaluated in fp32 from the fp32-rounded u, v and the integer
// radius so that it is reproducible bit for bit (SURVEY.md §8(c) reading A8).
inline void tile_rect_f32(float u, float v, int radius, int tile, int Gx, int Gy,
                          int& x0, int& x1, int& y0, int& y1) {
    const float inv = 1.0f / (float)tile;
    const float r_lo = (float)radius;
    const float r_hi = (float)(radius + tile - 1);
    auto clampi = [](int a, int lo, int hi) { return a < lo ? lo : (a > hi ? hi : a); };
    auto fl = [](float a) -> int {
        // floorf, then saturating conversion (values far outside the grid clamp anyway)
        float f = std::floor(a);
        if (!(f > -2.0e9f)) return -2000000000;
        if (!(f < 2.0e9f)) return 2000000000;
        return (int)f;
    };
    x0 = clampi(fl((u - r_lo) * inv), 0, Gx);
    x1 = clampi(fl((u + r_hi) * inv), 0, Gx);
    y0 = clampi(fl((v - r_lo) * inv), 0, Gy);
    y1 = clampi(fl((v + r_hi) * inv), 0, Gy);
}

// O-P1 steps 1, 3..8 for one Gaussian and one camera.
template <class R>
Proj<R> project_one(const Cfg& cfg, const Cam<R>& cam, const R p[3], const R Sig[3][3]) {
    Proj<R> o;
    o.visible = false; o.radius = 0; o.tiles = 0; o.radius_real = 0;
    // step 1
    for (int r = 0; r < 3; ++r) o.t[r] = cam.W[r][0] * p[0] + cam.W[r][1] * p[1] + cam.W[r][2] * p[2] + cam.tau[r];
    const R tz = o.t[2];
    if (!(tz > cam.near_plane) || !(tz < cam.far_plane)) return o;
    // step 3
    const R lim_x = (R)1.3 * (R)cam.width / (2 * cam.fx);
    const R lim_y = (R)1.3 * (R)cam.height / (2 * cam.fy);
    R rx = o.t[0] / tz, ry = o.t[1] / tz;
    o.clamp_x = (rx < -lim_x) || (rx > lim_x);
    o.clamp_y = (ry < -lim_y) || (ry > lim_y);
    rx = std::min(lim_x, std::max(-lim_x, rx));
    ry = std::min(lim_y, std::max(-lim_y, ry));
    o.xt = rx * tz; o.yt = ry * tz;
    o.J[0][0] = cam.fx / tz; o.J[0][1] = 0;           o.J[0][2] = -cam.fx * o.xt / (tz * tz);
    o.J[1][0] = 0;           o.J[1][1] = cam.fy / tz; o.J[1][2] = -cam.fy * o.yt / (tz * tz);
    // step 4
    for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 3; ++c) {
            R acc = 0;
            for (int k = 0; k < 3; ++k) acc += o.J[r][k] * cam.W[k][c];
            o.T[r][c] = acc;
        }
    R TS[2][3];
    for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 3; ++c) {
            R acc = 0;
            for (int k = 0; k < 3; ++k) acc += o.T[r][k] * Sig[k][c];
            TS[r][c] = acc;
        }
    R S2[2][2];
    for (int r = 0; r < 2; ++r)
        for (int c = 0; c < 2; ++c) {
            R acc = 0;
            for (int k = 0; k < 3; ++k) acc += TS[r][k] * o.T[c][k];
            S2[r][c] = acc;
        }
    o.a = S2[0][0] + (R)cfg.dilation;
    o.b = S2[0][1];
    o.c = S2[1][1] + (R)cfg.dilation;
    o.det = o.a * o.c - o.b * o.b;
    if (!(o.det > 0) || !std::isfinite(o.det)) return o;
    // step 5
    o.conic[0] = o.c / o.det; o.conic[1] = -o.b / o.det; o.conic[2] = o.a / o.det;
    // step 6
    const R m = (o.a + o.c) / 2;
    const R lam = m + std::sqrt(std::max((R)0.1, m * m - o.det));
    o.radius_real = (R)cfg.extent * std::sqrt(lam);
    const R rc = std::ceil(o.radius_real);
    if (!std::isfinite(rc)) return o;
    o.radius = rc > (R)1.0e9 ? 1000000000 : (int)rc;
    // step 7
    o.u = cam.fx * o.t[0] / tz + cam.cx;
    o.v = cam.fy * o.t[1] / tz + cam.cy;
    if (!std::isfinite(o.u) || !std::isfinite(o.v)) { o.radius = 0; return o; }
    // step 8
    const int Gx = (cam.width + cfg.tile - 1) / cfg.tile, Gy = (cam.height + cfg.tile - 1) / cfg.tile;
    tile_rect_f32((float)o.u, (float)o.v, o.radius, cfg.tile, Gx, Gy, o.x0, o.x1, o.y0, o.y1);
    o.tiles = (uint32_t)(o.x1 - o.x0) * (uint32_t)(o.y1 - o.y0);
    if (o.tiles == 0) { o.radius = 0; return o; }
    o.visible = true;
    return o;
}

// O-P1 step 9 helper: camera centre o = -W^T tau.
template <class R>
void cam_centre(const Cam<R>& cam, R o[3]) {
    for (int j = 0; j < 3; ++j) o[j] = -(cam.W[0][j] * cam.tau[0] + cam.W[1][j] * cam.tau[1] + cam.W[2][j] * cam.tau[2]);
}

// ---------------------------------------------------------------------------------------
// O-P1  gs_project_fwd  ("each GPU processes a segment of the input Gaussians
// and outputs colors and projected geometric quantities for all cameras in the batch")
// Outputs are laid out [C,N,*].  Culled entries: radius = 0, tiles_touched = 0, rest 0.
// ---------------------------------------------------------------------------------------
template <class R>
void project_fwd(const double* cfg_, int64_t N, const R* means, const R* log_scales, const R* quats,
                 const R* logits, const R* sh, int C, const double* cams_, R* means2d, R* depths, R* conics,
                 R* opacities, R* rgbs, int32_t* radii, uint32_t* tiles_touched, R* radius_real) {
    const Cfg cfg = load_cfg(cfg_);
    const int K = (cfg.deg + 1) * (cfg.deg + 1);
    for (int c = 0; c < C; ++c) {
        const Cam<R> cam = load_cam<R>(cams_ + 20 * c);
        R o[3];
        cam_centre(cam, o);
        for (int64_t i = 0; i < N; ++i) {
            const int64_t e = (int64_t)c * N + i;
            R s[3], qh[4], Rm[3][3], Mm[3][3], Sig[3][3];
            cov3d(log_scales + 3 * i, quats + 4 * i, s, qh, Rm, Mm, Sig);
            const Proj<R> pr = project_one(cfg, cam, means + 3 * i, Sig);
            radii[e] = pr.visible ? pr.radius : 0;
            tiles_touched[e] = pr.visible ? pr.tiles : 0;
            if (radius_real) radius_real[e] = pr.radius_real;
            if (!pr.visible) {
                means2d[2 * e] = means2d[2 * e + 1] = 0; depths[e] = 0;
                conics[3 * e] = conics[3 * e + 1] = conics[3 * e + 2] = 0;
                opacities[e] = 0; rgbs[3 * e] = rgbs[3 * e + 1] = rgbs[3 * e + 2] = 0;
                continue;
            }
            means2d[2 * e] = pr.u; means2d[2 * e + 1] = pr.v;
            depths[e] = pr.t[2];
            for (int k = 0; k < 3; ++k) conics[3 * e + k] = pr.conic[k];
            // step 9: colour
            R d[3] = {means[3 * i] - o[0], means[3 * i + 1] - o[1], means[3 * i + 2] - o[2]};
            const R dn = std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            R Y[16];
            sh_basis(d[0] / dn, d[1] / dn, d[2] / dn, Y);
            for (int ch = 0; ch < 3; ++ch) {
                R acc = 0;
                for (int k = 0; k < K; ++k) acc += Y[k] * sh[(i * K + k) * 3 + ch];
                acc += (R)0.5;
                rgbs[3 * e + ch] = acc > 0 ? acc : (R)0;
            }
            // step 10: opacity
            opacities[e] = 1 / (1 + std::exp(-logits[i]));
        }
    }
}

// ---------------------------------------------------------------------------------------
// O-R1  gs_raster_fwd  ("rasterizes them to obtain the rendered image";
// alpha rules = SURVEY.md §8(c) reading A11).  Views are batched: range index = c*tiles + t,
// isect_vals hold e = c*N + i into the [C,N,*] projected arrays.
// ambiguous (optional, [C,H,W] bytes): set when any decision came within rel_eps of its
// threshold (reading A17: several results are correct at decision boundaries).
// ---------------------------------------------------------------------------------------
template <class R>
void raster_fwd(const double* cfg_, int C, int width, int height, const int32_t* vals, const int64_t* ranges,
                const R* means2d, const R* conics, const R* opacities, const R* rgbs, const R* bg, R* image,
                R* final_T, int32_t* n_contrib, uint8_t* ambiguous, double rel_eps, const uint8_t* tile_mask) {
    const Cfg cfg = load_cfg(cfg_);
    const int Gx = (width + cfg.tile - 1) / cfg.tile, Gy = (height + cfg.tile - 1) / cfg.tile;
    const int64_t tiles = (int64_t)Gx * Gy;
    for (int c = 0; c < C; ++c)
        for (int i = 0; i < height; ++i)
            for (int j = 0; j < width; ++j) {
                const int64_t t = (int64_t)c * tiles + (int64_t)(i / cfg.tile) * Gx + (j / cfg.tile);
                if (tile_mask && !tile_mask[t]) continue;   // sampled evaluation: pixels of unselected tiles are left untouched
                const R px = (R)j + (R)0.5, py = (R)i + (R)0.5;
                R T = 1, Cacc[3] = {0, 0, 0};
                int32_t n = 0, last = 0;
                bool amb = false;
                for (int64_t k = ranges[2 * t]; k < ranges[2 * t + 1]; ++k) {
                    const int64_t g = vals[k];
                    ++n;
                    const R dx = means2d[2 * g] - px, dy = means2d[2 * g + 1] - py;
                    const R A = conics[3 * g], B = conics[3 * g + 1], Cc = conics[3 * g + 2];
                    const R power = -(R)0.5 * (A * dx * dx + Cc * dy * dy) - B * dx * dy;
                    if (ambiguous) {
                        const R mag = (R)0.5 * (std::fabs(A) * dx * dx + std::fabs(Cc) * dy * dy) + std::fabs(B * dx * dy);
                        if (std::fabs(power) <= (R)rel_eps * mag) amb = true;
                    }
                    if (power > 0) continue;
                    const R raw = opacities[g] * std::exp(power);
                    const R alpha = std::min((R)cfg.alpha_max, raw);
                    if (ambiguous && std::fabs(alpha - (R)cfg.alpha_min) <= (R)rel_eps * (R)cfg.alpha_min) amb = true;
                    if (alpha < (R)cfg.alpha_min) continue;
                    const R Tn = T * (1 - alpha);
                    if (ambiguous && std::fabs(Tn - (R)cfg.t_min) <= (R)rel_eps * (R)cfg.t_min) amb = true;
                    if (Tn < (R)cfg.t_min) break;
                    for (int ch = 0; ch < 3; ++ch) Cacc[ch] += rgbs[3 * g + ch] * alpha * T;
                    T = Tn;
                    last = n;
                }
                const int64_t pix = ((int64_t)c * height + i) * width + j;
                for (int ch = 0; ch < 3; ++ch) image[3 * pix + ch] = Cacc[ch] + T * bg[ch];
                final_T[pix] = T;
                n_contrib[pix] = last;
                if (ambiguous) ambiguous[pix] = amb ? 1 : 0;
            }
}

// ---------------------------------------------------------------------------------------
// O-R2  gs_raster_bwd  ("atomics are needed to accumulate gradients in the
// backward pass": here a plain sum).  Walk the first n_contrib entries backwards,
// re-evaluating the same skip tests; S = colour of everything behind the current entry.
// Outputs (size Ntot = C*N rows) are zeroed first.
// ---------------------------------------------------------------------------------------
template <class R>
void raster_bwd(const double* cfg_, int C, int width, int height, int64_t Ntot, const int32_t* vals,
                const int64_t* ranges, const R* means2d, const R* conics, const R* opacities, const R* rgbs,
                const R* bg, const R* final_T, const int32_t* n_contrib, const R* dL_dimage, R* dL_dmeans2d,
                R* dL_dconics, R* dL_dopacities, R* dL_drgbs, const uint8_t* tile_mask) {
    const Cfg cfg = load_cfg(cfg_);
    const int Gx = (width + cfg.tile - 1) / cfg.tile, Gy = (height + cfg.tile - 1) / cfg.tile;
    const int64_t tiles = (int64_t)Gx * Gy;
    std::fill(dL_dmeans2d, dL_dmeans2d + 2 * Ntot, (R)0);
    std::fill(dL_dconics, dL_dconics + 3 * Ntot, (R)0);
    std::fill(dL_dopacities, dL_dopacities + Ntot, (R)0);
    std::fill(dL_drgbs, dL_drgbs + 3 * Ntot, (R)0);
    for (int c = 0; c < C; ++c)
        for (int i = 0; i < height; ++i)
            for (int j = 0; j < width; ++j) {
                const int64_t t = (int64_t)c * tiles + (int64_t)(i / cfg.tile) * Gx + (j / cfg.tile);
                if (tile_mask && !tile_mask[t]) continue;   // sampled evaluation (caller zeroes dL_dimage there)
                const int64_t pix = ((int64_t)c * height + i) * width + j;
                const R px = (R)j + (R)0.5, py = (R)i + (R)0.5;
                const R* g3 = dL_dimage + 3 * pix;
                R T = final_T[pix];
                R S[3] = {bg[0], bg[1], bg[2]};
                const int64_t start = ranges[2 * t];
                for (int64_t k = start + n_contrib[pix] - 1; k >= start; --k) {
                    const int64_t g = vals[k];
                    const R dx = means2d[2 * g] - px, dy = means2d[2 * g + 1] - py;
                    const R A = conics[3 * g], B = conics[3 * g + 1], Cc = conics[3 * g + 2];
                    const R power = -(R)0.5 * (A * dx * dx + Cc * dy * dy) - B * dx * dy;
                    if (power > 0) continue;
                    const R G = std::exp(power);
                    const R raw = opacities[g] * G;
                    const R alpha = std::min((R)cfg.alpha_max, raw);
                    if (alpha < (R)cfg.alpha_min) continue;
                    // T_i: transmittance in front of entry i
                    T = T / (1 - alpha);
                    R dL_dalpha = 0;
                    for (int ch = 0; ch < 3; ++ch) {
                        dL_drgbs[3 * g + ch] += alpha * T * g3[ch];
                        dL_dalpha += T * (rgbs[3 * g + ch] - S[ch]) * g3[ch];
                    }
                    for (int ch = 0; ch < 3; ++ch) S[ch] = alpha * rgbs[3 * g + ch] + (1 - alpha) * S[ch];
                    if (raw > (R)cfg.alpha_max) continue;  // clamped: no gradient through alpha (reading A12)
                    dL_dopacities[g] += G * dL_dalpha;
                    const R dL_dpower = alpha * dL_dalpha;
                    dL_dconics[3 * g + 0] += -(R)0.5 * dx * dx * dL_dpower;
                    dL_dconics[3 * g + 1] += -dx * dy * dL_dpower;
                    dL_dconics[3 * g + 2] += -(R)0.5 * dy * dy * dL_dpower;
                    dL_dmeans2d[2 * g + 0] += -(A * dx + B * dy) * dL_dpower;
                    dL_dmeans2d[2 * g + 1] += -(B * dx + Cc * dy) * dL_dpower;
                }
            }
}

// ---------------------------------------------------------------------------------------
// O-P5  gs_project_bwd  (per-Gaussian partitioning, gradients summed over the
// views of the batch).  Chain rule of SURVEY.md §8(c) O-P5, written with small matrix loops.
// accumulate = 0: every row of every output is overwritten; 1: rows are added to.
// ---------------------------------------------------------------------------------------
template <class R>
void project_bwd(const double* cfg_, int64_t N, const R* means, const R* log_scales, const R* quats,
                 const R* logits, const R* sh, int C, const double* cams_, const int32_t* radii,
                 const R* g_means2d, const R* g_conics, const R* g_opacities, const R* g_rgbs, R* dL_dmeans,
                 R* dL_dlog_scales, R* dL_dquats, R* dL_dlogits, R* dL_dsh, int accumulate) {
    const Cfg cfg = load_cfg(cfg_);
    const int K = (cfg.deg + 1) * (cfg.deg + 1);
    std::vector<Cam<R>> cams;
    for (int c = 0; c < C; ++c) cams.push_back(load_cam<R>(cams_ + 20 * c));
    for (int64_t i = 0; i < N; ++i) {
        R gp[3] = {0, 0, 0}, gl[3] = {0, 0, 0}, gq[4] = {0, 0, 0, 0}, glogit = 0;
        std::vector<R> gsh((size_t)K * 3, (R)0);
        R s[3], qh[4], Rm[3][3], Mm[3][3], Sig[3][3];
        cov3d(log_scales + 3 * i, quats + 4 * i, s, qh, Rm, Mm, Sig);
        const R qn = std::sqrt(quats[4 * i] * quats[4 * i] + quats[4 * i + 1] * quats[4 * i + 1] +
                               quats[4 * i + 2] * quats[4 * i + 2] + quats[4 * i + 3] * quats[4 * i + 3]);
        const R op = 1 / (1 + std::exp(-logits[i]));
        for (int c = 0; c < C; ++c) {
            const int64_t e = (int64_t)c * N + i;
            if (radii[e] <= 0) continue;  // culled in this view: contributes nothing
            const Cam<R>& cam = cams[c];
            const Proj<R> pr = project_one(cfg, cam, means + 3 * i, Sig);
            if (!pr.visible) continue;
            const R tz = pr.t[2];
            // conic -> dilated 2-D covariance: G' = -K G_K K
            const R Kc[2][2] = {{pr.conic[0], pr.conic[1]}, {pr.conic[1], pr.conic[2]}};
            const R GK[2][2] = {{g_conics[3 * e], g_conics[3 * e + 1] / 2}, {g_conics[3 * e + 1] / 2, g_conics[3 * e + 2]}};
            R tmp[2][2], Gp[2][2];
            for (int r = 0; r < 2; ++r)
                for (int cc = 0; cc < 2; ++cc) tmp[r][cc] = Kc[r][0] * GK[0][cc] + Kc[r][1] * GK[1][cc];
            for (int r = 0; r < 2; ++r)
                for (int cc = 0; cc < 2; ++cc) Gp[r][cc] = -(tmp[r][0] * Kc[0][cc] + tmp[r][1] * Kc[1][cc]);
            // Sigma' = T Sigma T^T:  G_Sigma = T^T G' T,  G_T = 2 G' T Sigma
            R GpT[2][3];
            for (int r = 0; r < 2; ++r)
                for (int cc = 0; cc < 3; ++cc) GpT[r][cc] = Gp[r][0] * pr.T[0][cc] + Gp[r][1] * pr.T[1][cc];
            R GSig[3][3];
            for (int r = 0; r < 3; ++r)
                for (int cc = 0; cc < 3; ++cc) GSig[r][cc] = pr.T[0][r] * GpT[0][cc] + pr.T[1][r] * GpT[1][cc];
            R GT[2][3];
            for (int r = 0; r < 2; ++r)
                for (int cc = 0; cc < 3; ++cc) {
                    R acc = 0;
                    for (int k = 0; k < 3; ++k) acc += GpT[r][k] * Sig[k][cc];
                    GT[r][cc] = 2 * acc;
                }
            // T = J W:  G_J = G_T W^T
            R GJ[2][3];
            for (int r = 0; r < 2; ++r)
                for (int cc = 0; cc < 3; ++cc) {
                    R acc = 0;
                    for (int k = 0; k < 3; ++k) acc += GT[r][k] * cam.W[cc][k];
                    GJ[r][cc] = acc;
                }
            // dL/dt through mean2d (u = fx tx/tz + cx, v likewise; unclamped t)
            const R gu = g_means2d[2 * e], gv = g_means2d[2 * e + 1];
            R gt[3];
            gt[0] = gu * cam.fx / tz;
            gt[1] = gv * cam.fy / tz;
            gt[2] = -gu * cam.fx * pr.t[0] / (tz * tz) - gv * cam.fy * pr.t[1] / (tz * tz);
            // dL/dt through J (clamp of step 3: on a clamped axis J02 = -/+ fx lim / tz)
            const R tz2 = tz * tz, tz3 = tz2 * tz;
            gt[2] += -cam.fx / tz2 * GJ[0][0] - cam.fy / tz2 * GJ[1][1];
            if (pr.clamp_x) {
                gt[2] += cam.fx * pr.xt / tz3 * GJ[0][2];
            } else {
                gt[0] += -cam.fx / tz2 * GJ[0][2];
                gt[2] += 2 * cam.fx * pr.xt / tz3 * GJ[0][2];
            }
            if (pr.clamp_y) {
                gt[2] += cam.fy * pr.yt / tz3 * GJ[1][2];
            } else {
                gt[1] += -cam.fy / tz2 * GJ[1][2];
                gt[2] += 2 * cam.fy * pr.yt / tz3 * GJ[1][2];
            }
            // t = W p + tau
            for (int j = 0; j < 3; ++j) gp[j] += cam.W[0][j] * gt[0] + cam.W[1][j] * gt[1] + cam.W[2][j] * gt[2];
            // Sigma = M M^T:  G_M = 2 G_Sigma M;  M = R diag(s)
            R GM[3][3];
            for (int r = 0; r < 3; ++r)
                for (int k = 0; k < 3; ++k) {
                    R acc = 0;
                    for (int m = 0; m < 3; ++m) acc += GSig[r][m] * Mm[m][k];
                    GM[r][k] = 2 * acc;
                }
            R GR[3][3];
            for (int k = 0; k < 3; ++k) {
                R ds = 0;
                for (int r = 0; r < 3; ++r) ds += Rm[r][k] * GM[r][k];
                gl[k] += s[k] * ds;
                for (int r = 0; r < 3; ++r) GR[r][k] = GM[r][k] * s[k];
            }
            // R(q^) -> q^ -> q
            const R w = qh[0], x = qh[1], y = qh[2], z = qh[3];
            R gqh[4];
            gqh[0] = 2 * (x * (GR[2][1] - GR[1][2]) + y * (GR[0][2] - GR[2][0]) + z * (GR[1][0] - GR[0][1]));
            gqh[1] = 2 * (-2 * x * (GR[1][1] + GR[2][2]) + y * (GR[0][1] + GR[1][0]) + z * (GR[0][2] + GR[2][0]) + w * (GR[2][1] - GR[1][2]));
            gqh[2] = 2 * (x * (GR[0][1] + GR[1][0]) - 2 * y * (GR[0][0] + GR[2][2]) + z * (GR[1][2] + GR[2][1]) + w * (GR[0][2] - GR[2][0]));
            gqh[3] = 2 * (x * (GR[0][2] + GR[2][0]) + y * (GR[1][2] + GR[2][1]) - 2 * z * (GR[0][0] + GR[1][1]) + w * (GR[1][0] - GR[0][1]));
            const R dot = qh[0] * gqh[0] + qh[1] * gqh[1] + qh[2] * gqh[2] + qh[3] * gqh[3];
            for (int k = 0; k < 4; ++k) gq[k] += (gqh[k] - qh[k] * dot) / qn;
            // colour: rgb = max(0, sum_k Y_k(d^) f_k + 0.5)
            R o[3];
            cam_centre(cam, o);
            R d[3] = {means[3 * i] - o[0], means[3 * i + 1] - o[1], means[3 * i + 2] - o[2]};
            const R dn = std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            const R dh[3] = {d[0] / dn, d[1] / dn, d[2] / dn};
            R Y[16], dY[16][3];
            sh_basis(dh[0], dh[1], dh[2], Y);
            sh_basis_grad(dh[0], dh[1], dh[2], dY);
            R gdh[3] = {0, 0, 0};
            for (int ch = 0; ch < 3; ++ch) {
                R pre = 0;
                for (int k = 0; k < K; ++k) pre += Y[k] * sh[(i * K + k) * 3 + ch];
                pre += (R)0.5;
                if (!(pre > 0)) continue;  // clamped channel: gradient stops here
                const R gr = g_rgbs[3 * e + ch];
                for (int k = 0; k < K; ++k) {
                    gsh[(size_t)k * 3 + ch] += Y[k] * gr;
                    const R f = sh[(i * K + k) * 3 + ch];
                    for (int a = 0; a < 3; ++a) gdh[a] += dY[k][a] * f * gr;
                }
            }
            const R dd = dh[0] * gdh[0] + dh[1] * gdh[1] + dh[2] * gdh[2];
            for (int a = 0; a < 3; ++a) gp[a] += (gdh[a] - dh[a] * dd) / dn;
            // opacity = sigmoid(logit)
            glogit += op * (1 - op) * g_opacities[e];
        }
        if (accumulate) {
            for (int k = 0; k < 3; ++k) { dL_dmeans[3 * i + k] += gp[k]; dL_dlog_scales[3 * i + k] += gl[k]; }
            for (int k = 0; k < 4; ++k) dL_dquats[4 * i + k] += gq[k];
            dL_dlogits[i] += glogit;
            for (int k = 0; k < K * 3; ++k) dL_dsh[i * K * 3 + k] += gsh[k];
        } else {
            for (int k = 0; k < 3; ++k) { dL_dmeans[3 * i + k] = gp[k]; dL_dlog_scales[3 * i + k] = gl[k]; }
            for (int k = 0; k < 4; ++k) dL_dquats[4 * i + k] = gq[k];
            dL_dlogits[i] = glogit;
            for (int k = 0; k < K * 3; ++k) dL_dsh[i * K * 3 + k] = gsh[k];
        }
    }
}

}  // namespace

// =======================================================================================
// C entry points (host pointers everywhere)
// =======================================================================================
#define ORACLE_INSTANTIATE(SUF, R)                                                                              \
    extern "C" void oracle_project_fwd_##SUF(const double* cfg, int64_t N, const R* means, const R* log_scales, \
                                             const R* quats, const R* logits, const R* sh, int C,               \
                                             const double* cams, R* means2d, R* depths, R* conics,              \
                                             R* opacities, R* rgbs, int32_t* radii, uint32_t* tiles_touched,    \
                                             R* radius_real) {                                                  \
        project_fwd<R>(cfg, N, means, log_scales, quats, logits, sh, C, cams, means2d, depths, conics,          \
                       opacities, rgbs, radii, tiles_touched, radius_real);                                     \
    }                                                                                                           \
    extern "C" void oracle_raster_fwd_##SUF(const double* cfg, int C, int width, int height,                    \
                                            const int32_t* vals, const int64_t* ranges, const R* means2d,       \
                                            const R* conics, const R* opacities, const R* rgbs, const R* bg,    \
                                            R* image, R* final_T, int32_t* n_contrib, uint8_t* ambiguous,       \
                                            double rel_eps, const uint8_t* tile_mask) {                         \
        raster_fwd<R>(cfg, C, width, height, vals, ranges, means2d, conics, opacities, rgbs, bg, image,         \
                      final_T, n_contrib, ambiguous, rel_eps, tile_mask);                                       \
    }                                                                                                           \
    extern "C" void oracle_raster_bwd_##SUF(const double* cfg, int C, int width, int height, int64_t Ntot,      \
                                            const int32_t* vals, const int64_t* ranges, const R* means2d,       \
                                            const R* conics, const R* opacities, const R* rgbs, const R* bg,    \
                                            const R* final_T, const int32_t* n_contrib, const R* dL_dimage,     \
                                            R* dL_dmeans2d, R* dL_dconics, R* dL_dopacities, R* dL_drgbs,       \
                                            const uint8_t* tile_mask) {                                         \
        raster_bwd<R>(cfg, C, width, height, Ntot, vals, ranges, means2d, conics, opacities, rgbs, bg,          \
                      final_T, n_contrib, dL_dimage, dL_dmeans2d, dL_dconics, dL_dopacities, dL_drgbs,          \
                      tile_mask);                                                                               \
    }                                                                                                           \
    extern "C" void oracle_project_bwd_##SUF(const double* cfg, int64_t N, const R* means,                      \
                                             const R* log_scales, const R* quats, const R* logits,              \
                                             const R* sh, int C, const double* cams, const int32_t* radii,      \
                                             const R* g_means2d, const R* g_conics, const R* g_opacities,       \
                                             const R* g_rgbs, R* dL_dmeans, R* dL_dlog_scales, R* dL_dquats,    \
                                             R* dL_dlogits, R* dL_dsh, int accumulate) {                        \
        project_bwd<R>(cfg, N, means, log_scales, quats, logits, sh, C, cams, radii, g_means2d, g_conics,       \
                       g_opacities, g_rgbs, dL_dmeans, dL_dlog_scales, dL_dquats, dL_dlogits, dL_dsh,           \
                       accumulate);                                                                             \
    }                                                                                                           \
    extern "C" void oracle_sh_basis_##SUF(R x, R y, R z, R* Y16) { sh_basis<R>(x, y, z, Y16); }                 \
    extern "C" void oracle_cov3d_##SUF(const R* log_scale, const R* quat, R* Sigma9) {                          \
        R s[3], qh[4], Rm[3][3], Mm[3][3], Sig[3][3];                                                           \
        cov3d<R>(log_scale, quat, s, qh, Rm, Mm, Sig);                                                          \
        for (int r = 0; r < 3; ++r)                                                                             \
            for (int c = 0; c < 3; ++c) Sigma9[3 * r + c] = Sig[r][c];                                          \
    }

ORACLE_INSTANTIATE(f64, double)
ORACLE_INSTANTIATE(f32, float)

// ---------------------------------------------------------------------------------------
// O-B  gs_bin_tiles for a batch of C views ("the GPU sorts the Gaussians by
// depth"; "per-pixel/tile intersection records").  Integer / bit-level work,
// so it is not templated: inputs are the fp32 means2d and depths and the int32 radii.
//   offsets = exclusive prefix sum of tiles per (view, Gaussian) in (c, i) order
//   key = (uint64)(c*tiles + ty*Gx + tx) << 32 | bit_cast<uint32>(depth),  val = c*N + i
//   stable sort by key; ranges[t] = [first position with key>>32 == t, last + 1), [0,0) if none
// Returns M.  keys/vals may be NULL to query M only; capacity is checked by the caller.
// ---------------------------------------------------------------------------------------
extern "C" int64_t oracle_bin_tiles(const double* cfg_, int64_t N, int C, int width, int height,
                                    const float* means2d, const float* depths, const int32_t* radii,
                                    uint64_t* keys, int32_t* vals, int64_t* ranges) {
    const Cfg cfg = load_cfg(cfg_);
    const int Gx = (width + cfg.tile - 1) / cfg.tile, Gy = (height + cfg.tile - 1) / cfg.tile;
    const int64_t tiles = (int64_t)Gx * Gy;
    std::vector<std::pair<uint64_t, int32_t>> recs;
    int64_t M = 0;
    for (int c = 0; c < C; ++c)
        for (int64_t i = 0; i < N; ++i) {
            const int64_t e = (int64_t)c * N + i;
            if (radii[e] <= 0) continue;
            int x0, x1, y0, y1;
            tile_rect_f32(means2d[2 * e], means2d[2 * e + 1], radii[e], cfg.tile, Gx, Gy, x0, x1, y0, y1);
            uint32_t dbits;
            std::memcpy(&dbits, &depths[e], 4);
            for (int ty = y0; ty < y1; ++ty)
                for (int tx = x0; tx < x1; ++tx) {
                    if (keys) {
                        const uint64_t t = (uint64_t)c * (uint64_t)tiles + (uint64_t)ty * (uint64_t)Gx + (uint64_t)tx;
                        recs.emplace_back((t << 32) | (uint64_t)dbits, (int32_t)e);
                    }
                    ++M;
                }
        }
    if (!keys) return M;
    std::stable_sort(recs.begin(), recs.end(),
                     [](const std::pair<uint64_t, int32_t>& a, const std::pair<uint64_t, int32_t>& b) { return a.first < b.first; });
    for (int64_t t = 0; t < (int64_t)C * tiles; ++t) ranges[2 * t] = ranges[2 * t + 1] = 0;
    for (int64_t k = 0; k < M; ++k) {
        keys[k] = recs[k].first;
        vals[k] = recs[k].second;
        const int64_t t = (int64_t)(recs[k].first >> 32);
        if (k == 0 || (int64_t)(recs[k - 1].first >> 32) != t) ranges[2 * t] = k;
        ranges[2 * t + 1] = k + 1;
    }
    return M;
}
