// project_math.cuh -- per-Gaussian fp32 math of steps P1 / P5.
// Plain inline functions so the kernels in project.cu stay readable.
#pragma once

#include "common.cuh"

#if defined(__CUDACC__)
#define GS_HD __host__ __device__ __forceinline__
#else
#define GS_HD inline
#endif

namespace gs {

constexpr float kInfF = __builtin_huge_valf();

// Symmetric 3x3 stored as (xx, xy, xz, yy, yz, zz).
struct Sym3 {
    float xx, xy, xz, yy, yz, zz;
};

// O-P1 step 2: s = exp(l); q^ = q/|q| (w,x,y,z); R(q^); Sigma = R diag(s^2) R^T.
GS_HD void quat_rot(const float qh[4], float R[9]) {
    const float w = qh[0], x = qh[1], y = qh[2], z = qh[3];
    R[0] = 1.0f - 2.0f * (y * y + z * z); R[1] = 2.0f * (x * y - w * z);        R[2] = 2.0f * (x * z + w * y);
    R[3] = 2.0f * (x * y + w * z);        R[4] = 1.0f - 2.0f * (x * x + z * z); R[5] = 2.0f * (y * z - w * x);
    R[6] = 2.0f * (x * z - w * y);        R[7] = 2.0f * (y * z + w * x);        R[8] = 1.0f - 2.0f * (x * x + y * y);
}
GS_HD void cov3d(const float ls[3], const float q[4], float s[3], float qh[4], float& qnorm, float R[9], Sym3& S) {
    s[0] = expf(ls[0]); s[1] = expf(ls[1]); s[2] = expf(ls[2]);
    qnorm = sqrtf(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    const float inv = 1.0f / qnorm;
    qh[0] = q[0] * inv; qh[1] = q[1] * inv; qh[2] = q[2] * inv; qh[3] = q[3] * inv;
    quat_rot(qh, R);
    const float s0 = s[0] * s[0], s1 = s[1] * s[1], s2 = s[2] * s[2];
    S.xx = R[0] * R[0] * s0 + R[1] * R[1] * s1 + R[2] * R[2] * s2;
    S.xy = R[0] * R[3] * s0 + R[1] * R[4] * s1 + R[2] * R[5] * s2;
    S.xz = R[0] * R[6] * s0 + R[1] * R[7] * s1 + R[2] * R[8] * s2;
    S.yy = R[3] * R[3] * s0 + R[4] * R[4] * s1 + R[5] * R[5] * s2;
    S.yz = R[3] * R[6] * s0 + R[4] * R[7] * s1 + R[5] * R[8] * s2;
    S.zz = R[6] * R[6] * s0 + R[7] * R[7] * s1 + R[8] * R[8] * s2;
}

// Intermediates of O-P1 steps 1, 3, 4 that the backward pass needs again.
struct ProjMid {
    float tx, ty, tz, rz;      // camera-space mean, 1/tz
    float rxc, ryc;            // clamped tx/tz, ty/tz
    bool clamp_x, clamp_y;
    float T0[3], T1[3];        // rows of T = J W
    float a, b, c, det;        // dilated 2-D covariance
};

// Steps 1, 3, 4.  Returns false when culled by near/far or det.
GS_HD bool project_mid(const DevCam& cam, float px, float py, float pz, const Sym3& S, float dilation, ProjMid& m) {
    m.tx = cam.W[0] * px + cam.W[1] * py + cam.W[2] * pz + cam.tau[0];
    m.ty = cam.W[3] * px + cam.W[4] * py + cam.W[5] * pz + cam.tau[1];
    m.tz = cam.W[6] * px + cam.W[7] * py + cam.W[8] * pz + cam.tau[2];
    if (!(m.tz > cam.near_plane) || !(m.tz < cam.far_plane)) return false;
    m.rz = 1.0f / m.tz;
    const float rx = m.tx * m.rz, ry = m.ty * m.rz;
    m.clamp_x = (rx < -cam.lim_x) || (rx > cam.lim_x);
    m.clamp_y = (ry < -cam.lim_y) || (ry > cam.lim_y);
    m.rxc = fminf(cam.lim_x, fmaxf(-cam.lim_x, rx));
    m.ryc = fminf(cam.lim_y, fmaxf(-cam.lim_y, ry));
    // J = [[fx/tz, 0, -fx x~/tz^2], [0, fy/tz, -fy y~/tz^2]] with x~/tz = rxc
    const float j00 = cam.fx * m.rz, j02 = -cam.fx * m.rxc * m.rz;
    const float j11 = cam.fy * m.rz, j12 = -cam.fy * m.ryc * m.rz;
    for (int k = 0; k < 3; ++k) {
        m.T0[k] = j00 * cam.W[k] + j02 * cam.W[6 + k];
        m.T1[k] = j11 * cam.W[3 + k] + j12 * cam.W[6 + k];
    }
    // Sigma' = T Sigma T^T
    const float v0x = S.xx * m.T0[0] + S.xy * m.T0[1] + S.xz * m.T0[2];
    const float v0y = S.xy * m.T0[0] + S.yy * m.T0[1] + S.yz * m.T0[2];
    const float v0z = S.xz * m.T0[0] + S.yz * m.T0[1] + S.zz * m.T0[2];
    const float v1x = S.xx * m.T1[0] + S.xy * m.T1[1] + S.xz * m.T1[2];
    const float v1y = S.xy * m.T1[0] + S.yy * m.T1[1] + S.yz * m.T1[2];
    const float v1z = S.xz * m.T1[0] + S.yz * m.T1[1] + S.zz * m.T1[2];
    m.a = m.T0[0] * v0x + m.T0[1] * v0y + m.T0[2] * v0z + dilation;
    m.b = m.T1[0] * v0x + m.T1[1] * v0y + m.T1[2] * v0z;
    m.c = m.T1[0] * v1x + m.T1[1] * v1y + m.T1[2] * v1z + dilation;
    m.det = m.a * m.c - m.b * m.b;
    if (!(m.det > 0.0f) || !(m.det < kInfF)) return false;
    return true;
}

// Real SH basis (degrees 0..DEG) at unit direction (x,y,z).
template <int DEG>
GS_HD void sh_basis(float x, float y, float z, float* Y) {
    Y[0] = kC0;
    if (DEG >= 1) {
        Y[1] = -kC1 * y; Y[2] = kC1 * z; Y[3] = -kC1 * x;
    }
    if (DEG >= 2) {
        const float xx = x * x, yy = y * y, zz = z * z;
        Y[4] = kC2a * x * y;
        Y[5] = -kC2a * y * z;
        Y[6] = kC2b * (2.0f * zz - xx - yy);
        Y[7] = -kC2a * x * z;
        Y[8] = kC2c * (xx - yy);
        if (DEG >= 3) {
            Y[9] = -kC3a * y * (3.0f * xx - yy);
            Y[10] = kC3b * x * y * z;
            Y[11] = -kC3c * y * (4.0f * zz - xx - yy);
            Y[12] = kC3d * z * (2.0f * zz - 3.0f * xx - 3.0f * yy);
            Y[13] = -kC3c * x * (4.0f * zz - xx - yy);
            Y[14] = kC3e * z * (xx - yy);
            Y[15] = -kC3a * x * (xx - 3.0f * yy);
        }
    }
}

// d/d(x,y,z) of every basis polynomial (unconstrained); dY[k] = (dx, dy, dz).
template <int DEG>
GS_HD void sh_basis_grad(float x, float y, float z, float (*dY)[3]) {
    dY[0][0] = 0.f; dY[0][1] = 0.f; dY[0][2] = 0.f;
    if (DEG >= 1) {
        dY[1][0] = 0.f;   dY[1][1] = -kC1; dY[1][2] = 0.f;
        dY[2][0] = 0.f;   dY[2][1] = 0.f;  dY[2][2] = kC1;
        dY[3][0] = -kC1;  dY[3][1] = 0.f;  dY[3][2] = 0.f;
    }
    if (DEG >= 2) {
        dY[4][0] = kC2a * y;         dY[4][1] = kC2a * x;         dY[4][2] = 0.f;
        dY[5][0] = 0.f;              dY[5][1] = -kC2a * z;        dY[5][2] = -kC2a * y;
        dY[6][0] = -2.0f * kC2b * x; dY[6][1] = -2.0f * kC2b * y; dY[6][2] = 4.0f * kC2b * z;
        dY[7][0] = -kC2a * z;        dY[7][1] = 0.f;              dY[7][2] = -kC2a * x;
        dY[8][0] = 2.0f * kC2c * x;  dY[8][1] = -2.0f * kC2c * y; dY[8][2] = 0.f;
    }
    if (DEG >= 3) {
        const float xx = x * x, yy = y * y, zz = z * z;
        dY[9][0] = -6.0f * kC3a * x * y;           dY[9][1] = -3.0f * kC3a * (xx - yy);           dY[9][2] = 0.f;
        dY[10][0] = kC3b * y * z;                  dY[10][1] = kC3b * x * z;                      dY[10][2] = kC3b * x * y;
        dY[11][0] = 2.0f * kC3c * x * y;           dY[11][1] = -kC3c * (4.0f * zz - xx - 3.0f * yy); dY[11][2] = -8.0f * kC3c * y * z;
        dY[12][0] = -6.0f * kC3d * x * z;          dY[12][1] = -6.0f * kC3d * y * z;              dY[12][2] = 3.0f * kC3d * (2.0f * zz - xx - yy);
        dY[13][0] = -kC3c * (4.0f * zz - 3.0f * xx - yy); dY[13][1] = 2.0f * kC3c * x * y;        dY[13][2] = -8.0f * kC3c * x * z;
        dY[14][0] = 2.0f * kC3e * x * z;           dY[14][1] = -2.0f * kC3e * y * z;              dY[14][2] = kC3e * (xx - yy);
        dY[15][0] = -3.0f * kC3a * (xx - yy);      dY[15][1] = 6.0f * kC3a * x * y;               dY[15][2] = 0.f;
    }
}

}  // namespace gs
