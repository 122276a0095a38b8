// project.cu -- per-Gaussian stages P1 (gs_project_fwd) and P5 (gs_project_bwd) for sm_100a.
//
// One thread per Gaussian; the C views of the batch are looped inside the thread so that the
// parameters (236 B at SH degree 3) are read once for all cameras ("outputs colors
// and projected geometric quantities for all cameras in the batch").  Culling happens on the
// 12-byte mean first; scale/rotation are read only for Gaussians inside some view's depth range
// and the SH coefficients only for Gaussians visible in at least one view, so the HBM traffic is
// 12 N + 224 V_any + 48 sum_c V_c + 8 N C ("algorithmic bytes").
#include "project_math.cuh"

namespace gs {

struct ProjFwdArgs {
    int64_t N;
    int32_t C;
    const float* means; const float* log_scales; const float* quats; const float* logits; const float* sh;
    float* means2d; float* depths; float* conics; float* opacities; float* rgbs;
    int32_t* radii; uint32_t* tiles;
    float dilation, extent;
};

constexpr int kProjThreads = 128;

template <int DEG>
__device__ __forceinline__ void load_sh(const float* __restrict__ sh, int64_t i, float* f) {
    constexpr int K3 = 3 * (DEG + 1) * (DEG + 1);
    const float* p = sh + i * K3;
    if constexpr (K3 % 4 == 0) {
        const float4* p4 = reinterpret_cast<const float4*>(p);
#pragma unroll
        for (int k = 0; k < K3 / 4; ++k) {
            const float4 v = __ldg(p4 + k);
            f[4 * k] = v.x; f[4 * k + 1] = v.y; f[4 * k + 2] = v.z; f[4 * k + 3] = v.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < K3; ++k) f[k] = __ldg(p + k);
    }
}

template <int DEG>
__global__ void __launch_bounds__(kProjThreads) project_fwd_kernel(const ProjFwdArgs a, const __grid_constant__ CamBatch cams) {
    const int64_t i = (int64_t)blockIdx.x * kProjThreads + threadIdx.x;
    if (i >= a.N) return;
    const float px = __ldg(a.means + 3 * i), py = __ldg(a.means + 3 * i + 1), pz = __ldg(a.means + 3 * i + 2);

    // depth-range test on the mean alone (step 1)
    uint32_t zmask = 0;
    for (int c = 0; c < a.C; ++c) {
        const DevCam& cam = cams.cam[c];
        const float tz = cam.W[6] * px + cam.W[7] * py + cam.W[8] * pz + cam.tau[2];
        if (tz > cam.near_plane && tz < cam.far_plane) zmask |= 1u << c;
    }
    uint32_t vis = 0;
    if (zmask) {
        float ls[3], q[4], s[3], qh[4], qn, R[9];
        Sym3 S;
        ls[0] = __ldg(a.log_scales + 3 * i); ls[1] = __ldg(a.log_scales + 3 * i + 1); ls[2] = __ldg(a.log_scales + 3 * i + 2);
        const float4 qv = __ldg(reinterpret_cast<const float4*>(a.quats) + i);
        q[0] = qv.x; q[1] = qv.y; q[2] = qv.z; q[3] = qv.w;
        cov3d(ls, q, s, qh, qn, R, S);
        for (int c = 0; c < a.C; ++c) {
            if (!((zmask >> c) & 1u)) continue;
            const DevCam& cam = cams.cam[c];
            ProjMid m;
            if (!project_mid(cam, px, py, pz, S, a.dilation, m)) continue;
            // step 6: radius from the larger eigenvalue
            const float mid = 0.5f * (m.a + m.c);
            const float lam = mid + sqrtf(fmaxf(0.1f, mid * mid - m.det));
            const float rr = ceilf(a.extent * sqrtf(lam));
            if (!(rr < kInfF)) continue;
            const int radius = (int)fminf(rr, 1.0e9f);
            // step 7
            const float u = cam.fx * m.tx * m.rz + cam.cx;
            const float v = cam.fy * m.ty * m.rz + cam.cy;
            if (!(fabsf(u) < kInfF) || !(fabsf(v) < kInfF)) continue;
            // step 8
            int x0, x1, y0, y1;
            tile_rect(u, v, radius, cam.gx, cam.gy, x0, x1, y0, y1);
            const uint32_t nt = (uint32_t)(x1 - x0) * (uint32_t)(y1 - y0);
            if (nt == 0) continue;
            vis |= 1u << c;
            const int64_t e = (int64_t)c * a.N + i;
            const float inv = 1.0f / m.det;
            reinterpret_cast<float2*>(a.means2d)[e] = make_float2(u, v);
            a.depths[e] = m.tz;
            a.conics[3 * e] = m.c * inv; a.conics[3 * e + 1] = -m.b * inv; a.conics[3 * e + 2] = m.a * inv;
            a.radii[e] = radius;
            a.tiles[e] = nt;
        }
    }
    for (int c = 0; c < a.C; ++c)
        if (!((vis >> c) & 1u)) {
            const int64_t e = (int64_t)c * a.N + i;
            a.radii[e] = 0;
            a.tiles[e] = 0;
        }
    if (!vis) return;

    // steps 9, 10: colour and opacity, only for Gaussians visible somewhere
    constexpr int K = (DEG + 1) * (DEG + 1);
    float f[3 * K];
    load_sh<DEG>(a.sh, i, f);
    const float opacity = 1.0f / (1.0f + expf(-__ldg(a.logits + i)));
    for (int c = 0; c < a.C; ++c) {
        if (!((vis >> c) & 1u)) continue;
        const DevCam& cam = cams.cam[c];
        const float dx = px - cam.ox, dy = py - cam.oy, dz = pz - cam.oz;
        const float dinv = 1.0f / sqrtf(dx * dx + dy * dy + dz * dz);
        float Y[K];
        sh_basis<DEG>(dx * dinv, dy * dinv, dz * dinv, Y);
        float r = 0.5f, g = 0.5f, b = 0.5f;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            r = fmaf(Y[k], f[3 * k], r);
            g = fmaf(Y[k], f[3 * k + 1], g);
            b = fmaf(Y[k], f[3 * k + 2], b);
        }
        const int64_t e = (int64_t)c * a.N + i;
        a.rgbs[3 * e] = fmaxf(r, 0.0f); a.rgbs[3 * e + 1] = fmaxf(g, 0.0f); a.rgbs[3 * e + 2] = fmaxf(b, 0.0f);
        a.opacities[e] = opacity;
    }
}

// ---------------------------------------------------------------------------------------------
struct ProjBwdArgs {
    int64_t N;
    int32_t C;
    const float* means; const float* log_scales; const float* quats; const float* logits; const float* sh;
    const int32_t* radii;
    const float* g_means2d; const float* g_conics; const float* g_opacities; const float* g_rgbs;
    float* d_means; float* d_log_scales; float* d_quats; float* d_logits; float* d_sh;
    float dilation;
    int32_t accumulate;
};

template <int DEG>
__device__ __forceinline__ void store_sh(float* __restrict__ out, int64_t i, const float* g, bool accumulate) {
    constexpr int K3 = 3 * (DEG + 1) * (DEG + 1);
    float* p = out + i * K3;
    if constexpr (K3 % 4 == 0) {
        float4* p4 = reinterpret_cast<float4*>(p);
#pragma unroll
        for (int k = 0; k < K3 / 4; ++k) {
            float4 v = make_float4(g[4 * k], g[4 * k + 1], g[4 * k + 2], g[4 * k + 3]);
            if (accumulate) {
                const float4 o = p4[k];
                v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w;
            }
            p4[k] = v;
        }
    } else {
#pragma unroll
        for (int k = 0; k < K3; ++k) p[k] = accumulate ? p[k] + g[k] : g[k];
    }
}

template <int DEG>
__global__ void __launch_bounds__(kProjThreads) project_bwd_kernel(const ProjBwdArgs a, const __grid_constant__ CamBatch cams) {
    const int64_t i = (int64_t)blockIdx.x * kProjThreads + threadIdx.x;
    if (i >= a.N) return;
    constexpr int K = (DEG + 1) * (DEG + 1);

    uint32_t vis = 0;
    for (int c = 0; c < a.C; ++c)
        if (__ldg(a.radii + (int64_t)c * a.N + i) > 0) vis |= 1u << c;

    float gp[3] = {0.f, 0.f, 0.f}, gl[3] = {0.f, 0.f, 0.f}, gq[4] = {0.f, 0.f, 0.f, 0.f}, glogit = 0.f;
    float gsh[3 * K];
#pragma unroll
    for (int k = 0; k < 3 * K; ++k) gsh[k] = 0.f;

    if (vis) {
        const float px = __ldg(a.means + 3 * i), py = __ldg(a.means + 3 * i + 1), pz = __ldg(a.means + 3 * i + 2);
        float ls[3], q[4], s[3], qh[4], qn, R[9];
        Sym3 S;
        ls[0] = __ldg(a.log_scales + 3 * i); ls[1] = __ldg(a.log_scales + 3 * i + 1); ls[2] = __ldg(a.log_scales + 3 * i + 2);
        const float4 qv = __ldg(reinterpret_cast<const float4*>(a.quats) + i);
        q[0] = qv.x; q[1] = qv.y; q[2] = qv.z; q[3] = qv.w;
        cov3d(ls, q, s, qh, qn, R, S);
        float f[3 * K];
        load_sh<DEG>(a.sh, i, f);
        // gradient with respect to Sigma, summed over views (full symmetric matrix, 6 unique entries)
        float Gxx = 0.f, Gxy = 0.f, Gxz = 0.f, Gyy = 0.f, Gyz = 0.f, Gzz = 0.f;
        float g_op = 0.f;
        for (int c = 0; c < a.C; ++c) {
            if (!((vis >> c) & 1u)) continue;
            const DevCam& cam = cams.cam[c];
            ProjMid m;
            if (!project_mid(cam, px, py, pz, S, a.dilation, m)) continue;
            const int64_t e = (int64_t)c * a.N + i;
            const float2 guv = __ldg(reinterpret_cast<const float2*>(a.g_means2d) + e);
            const float gA = __ldg(a.g_conics + 3 * e), gB = __ldg(a.g_conics + 3 * e + 1), gC = __ldg(a.g_conics + 3 * e + 2);
            g_op += __ldg(a.g_opacities + e);
            // conic -> dilated covariance: G' = -K G_K K
            const float inv = 1.0f / m.det;
            const float A = m.c * inv, B = -m.b * inv, Cc = m.a * inv;
            const float h = 0.5f * gB;
            const float t00 = A * gA + B * h, t01 = A * h + B * gC;
            const float t10 = B * gA + Cc * h, t11 = B * h + Cc * gC;
            const float P00 = -(t00 * A + t01 * B);
            const float P01 = -(t00 * B + t01 * Cc);
            const float P11 = -(t10 * B + t11 * Cc);
            // G_Sigma += T^T G' T
            const float* T0 = m.T0; const float* T1 = m.T1;
            Gxx += P00 * T0[0] * T0[0] + 2.0f * P01 * T0[0] * T1[0] + P11 * T1[0] * T1[0];
            Gyy += P00 * T0[1] * T0[1] + 2.0f * P01 * T0[1] * T1[1] + P11 * T1[1] * T1[1];
            Gzz += P00 * T0[2] * T0[2] + 2.0f * P01 * T0[2] * T1[2] + P11 * T1[2] * T1[2];
            Gxy += P00 * T0[0] * T0[1] + P01 * (T0[0] * T1[1] + T1[0] * T0[1]) + P11 * T1[0] * T1[1];
            Gxz += P00 * T0[0] * T0[2] + P01 * (T0[0] * T1[2] + T1[0] * T0[2]) + P11 * T1[0] * T1[2];
            Gyz += P00 * T0[1] * T0[2] + P01 * (T0[1] * T1[2] + T1[1] * T0[2]) + P11 * T1[1] * T1[2];
            // G_T = 2 G' T Sigma ; G_J = G_T W^T (only the four live entries of J)
            const float v0x = S.xx * T0[0] + S.xy * T0[1] + S.xz * T0[2];
            const float v0y = S.xy * T0[0] + S.yy * T0[1] + S.yz * T0[2];
            const float v0z = S.xz * T0[0] + S.yz * T0[1] + S.zz * T0[2];
            const float v1x = S.xx * T1[0] + S.xy * T1[1] + S.xz * T1[2];
            const float v1y = S.xy * T1[0] + S.yy * T1[1] + S.yz * T1[2];
            const float v1z = S.xz * T1[0] + S.yz * T1[1] + S.zz * T1[2];
            const float GT0x = 2.0f * (P00 * v0x + P01 * v1x), GT0y = 2.0f * (P00 * v0y + P01 * v1y), GT0z = 2.0f * (P00 * v0z + P01 * v1z);
            const float GT1x = 2.0f * (P01 * v0x + P11 * v1x), GT1y = 2.0f * (P01 * v0y + P11 * v1y), GT1z = 2.0f * (P01 * v0z + P11 * v1z);
            const float GJ00 = GT0x * cam.W[0] + GT0y * cam.W[1] + GT0z * cam.W[2];
            const float GJ02 = GT0x * cam.W[6] + GT0y * cam.W[7] + GT0z * cam.W[8];
            const float GJ11 = GT1x * cam.W[3] + GT1y * cam.W[4] + GT1z * cam.W[5];
            const float GJ12 = GT1x * cam.W[6] + GT1y * cam.W[7] + GT1z * cam.W[8];
            // dL/dt through mean2d and through J (clamped axes: J02 = -/+ fx lim / tz)
            const float rz2 = m.rz * m.rz;
            float gtx = guv.x * cam.fx * m.rz;
            float gty = guv.y * cam.fy * m.rz;
            float gtz = -(guv.x * cam.fx * m.tx + guv.y * cam.fy * m.ty) * rz2;
            gtz -= (cam.fx * GJ00 + cam.fy * GJ11) * rz2;
            const float kx = cam.fx * m.rxc * rz2, ky = cam.fy * m.ryc * rz2;
            if (m.clamp_x) {
                gtz += kx * GJ02;
            } else {
                gtx -= cam.fx * rz2 * GJ02;
                gtz += 2.0f * kx * GJ02;
            }
            if (m.clamp_y) {
                gtz += ky * GJ12;
            } else {
                gty -= cam.fy * rz2 * GJ12;
                gtz += 2.0f * ky * GJ12;
            }
            gp[0] += cam.W[0] * gtx + cam.W[3] * gty + cam.W[6] * gtz;
            gp[1] += cam.W[1] * gtx + cam.W[4] * gty + cam.W[7] * gtz;
            gp[2] += cam.W[2] * gtx + cam.W[5] * gty + cam.W[8] * gtz;
            // colour
            const float dx = px - cam.ox, dy = py - cam.oy, dz = pz - cam.oz;
            const float dinv = 1.0f / sqrtf(dx * dx + dy * dy + dz * dz);
            const float hx = dx * dinv, hy = dy * dinv, hz = dz * dinv;
            float Y[K];
            sh_basis<DEG>(hx, hy, hz, Y);
            float pre[3] = {0.5f, 0.5f, 0.5f};
#pragma unroll
            for (int k = 0; k < K; ++k) {
                pre[0] = fmaf(Y[k], f[3 * k], pre[0]);
                pre[1] = fmaf(Y[k], f[3 * k + 1], pre[1]);
                pre[2] = fmaf(Y[k], f[3 * k + 2], pre[2]);
            }
            float gr[3];
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) gr[ch] = pre[ch] > 0.0f ? __ldg(a.g_rgbs + 3 * e + ch) : 0.0f;
            float gh[3] = {0.f, 0.f, 0.f};
            if (DEG >= 1) {
                float dY[K][3];
                sh_basis_grad<DEG>(hx, hy, hz, dY);
#pragma unroll
                for (int k = 1; k < K; ++k) {
                    const float vk = f[3 * k] * gr[0] + f[3 * k + 1] * gr[1] + f[3 * k + 2] * gr[2];
                    gh[0] = fmaf(dY[k][0], vk, gh[0]);
                    gh[1] = fmaf(dY[k][1], vk, gh[1]);
                    gh[2] = fmaf(dY[k][2], vk, gh[2]);
                }
                const float dd = hx * gh[0] + hy * gh[1] + hz * gh[2];
                gp[0] += (gh[0] - hx * dd) * dinv;
                gp[1] += (gh[1] - hy * dd) * dinv;
                gp[2] += (gh[2] - hz * dd) * dinv;
            }
#pragma unroll
            for (int k = 0; k < K; ++k) {
                gsh[3 * k] = fmaf(Y[k], gr[0], gsh[3 * k]);
                gsh[3 * k + 1] = fmaf(Y[k], gr[1], gsh[3 * k + 1]);
                gsh[3 * k + 2] = fmaf(Y[k], gr[2], gsh[3 * k + 2]);
            }
        }
        // Sigma = M M^T, M = R diag(s):  G_M = 2 G_Sigma M
        const float G[9] = {Gxx, Gxy, Gxz, Gxy, Gyy, Gyz, Gxz, Gyz, Gzz};
        float GR[9];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            float ds = 0.f;
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                const float gm = 2.0f * s[k] * (G[3 * r] * R[k] + G[3 * r + 1] * R[3 + k] + G[3 * r + 2] * R[6 + k]);
                ds = fmaf(R[3 * r + k], gm, ds);
                GR[3 * r + k] = gm * s[k];
            }
            gl[k] = s[k] * ds;
        }
        // R(q^) -> q^ -> q
        const float w = qh[0], x = qh[1], y = qh[2], z = qh[3];
        float gh4[4];
        gh4[0] = 2.0f * (x * (GR[7] - GR[5]) + y * (GR[2] - GR[6]) + z * (GR[3] - GR[1]));
        gh4[1] = 2.0f * (-2.0f * x * (GR[4] + GR[8]) + y * (GR[1] + GR[3]) + z * (GR[2] + GR[6]) + w * (GR[7] - GR[5]));
        gh4[2] = 2.0f * (x * (GR[1] + GR[3]) - 2.0f * y * (GR[0] + GR[8]) + z * (GR[5] + GR[7]) + w * (GR[2] - GR[6]));
        gh4[3] = 2.0f * (x * (GR[2] + GR[6]) + y * (GR[5] + GR[7]) - 2.0f * z * (GR[0] + GR[4]) + w * (GR[3] - GR[1]));
        const float dot = w * gh4[0] + x * gh4[1] + y * gh4[2] + z * gh4[3];
        const float qinv = 1.0f / qn;
#pragma unroll
        for (int k = 0; k < 4; ++k) gq[k] = (gh4[k] - qh[k] * dot) * qinv;
        const float op = 1.0f / (1.0f + expf(-__ldg(a.logits + i)));
        glogit = op * (1.0f - op) * g_op;
    }

    if (a.accumulate) {
        if (!vis) return;
#pragma unroll
        for (int k = 0; k < 3; ++k) { a.d_means[3 * i + k] += gp[k]; a.d_log_scales[3 * i + k] += gl[k]; }
        float4* dq = reinterpret_cast<float4*>(a.d_quats) + i;
        float4 o = *dq;
        o.x += gq[0]; o.y += gq[1]; o.z += gq[2]; o.w += gq[3];
        *dq = o;
        a.d_logits[i] += glogit;
        store_sh<DEG>(a.d_sh, i, gsh, true);
    } else {
#pragma unroll
        for (int k = 0; k < 3; ++k) { a.d_means[3 * i + k] = gp[k]; a.d_log_scales[3 * i + k] = gl[k]; }
        reinterpret_cast<float4*>(a.d_quats)[i] = make_float4(gq[0], gq[1], gq[2], gq[3]);
        a.d_logits[i] = glogit;
        store_sh<DEG>(a.d_sh, i, gsh, false);
    }
}

template <int DEG>
int launch_fwd(const ProjFwdArgs& a, const CamBatch& cb, cudaStream_t st) {
    const int64_t blocks = (a.N + kProjThreads - 1) / kProjThreads;
    project_fwd_kernel<DEG><<<(unsigned)blocks, kProjThreads, 0, st>>>(a, cb);
    return launch_status();
}
template <int DEG>
int launch_bwd(const ProjBwdArgs& a, const CamBatch& cb, cudaStream_t st) {
    const int64_t blocks = (a.N + kProjThreads - 1) / kProjThreads;
    project_bwd_kernel<DEG><<<(unsigned)blocks, kProjThreads, 0, st>>>(a, cb);
    return launch_status();
}

}  // namespace gs

using namespace gs;

extern "C" int gs_project_fwd(const gs_config* cfg, int64_t N, const float* means, const float* log_scales,
                              const float* quats, const float* opacity_logits, const float* sh, int32_t C,
                              const gs_camera* cams, float* means2d, float* depths, float* conics, float* opacities,
                              float* rgbs, int32_t* radii, uint32_t* tiles_touched, void* stream) {
    int rc = check_cfg(cfg);
    if (rc) return rc;
    rc = check_cams(C, cams);
    if (rc) return rc;
    if (N < 0) return GS_ERR_INVALID_ARGUMENT;
    if (N == 0) return GS_OK;
    if (!means || !log_scales || !quats || !opacity_logits || !sh || !means2d || !depths || !conics || !opacities ||
        !rgbs || !radii || !tiles_touched)
        return GS_ERR_INVALID_ARGUMENT;
    if (!aligned(quats, 16) || !aligned(sh, 16) || !aligned(means2d, 8) || !aligned(means, 4)) return GS_ERR_INVALID_ARGUMENT;
    if ((N + kProjThreads - 1) / kProjThreads > 0x7fffffffLL || (int64_t)C * N >= (1LL << 31)) return GS_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    for (int c0 = 0; c0 < C; c0 += kMaxCamsPerLaunch) {
        const int nc = C - c0 < kMaxCamsPerLaunch ? C - c0 : kMaxCamsPerLaunch;
        CamBatch cb;
        for (int c = 0; c < nc; ++c) cb.cam[c] = make_devcam(cams[c0 + c]);
        ProjFwdArgs a;
        a.N = N; a.C = nc;
        a.means = means; a.log_scales = log_scales; a.quats = quats; a.logits = opacity_logits; a.sh = sh;
        const int64_t off = (int64_t)c0 * N;
        a.means2d = means2d + 2 * off; a.depths = depths + off; a.conics = conics + 3 * off;
        a.opacities = opacities + off; a.rgbs = rgbs + 3 * off; a.radii = radii + off; a.tiles = tiles_touched + off;
        a.dilation = cfg->dilation; a.extent = cfg->extent;
        switch (cfg->sh_degree) {
            case 0: rc = launch_fwd<0>(a, cb, st); break;
            case 1: rc = launch_fwd<1>(a, cb, st); break;
            case 2: rc = launch_fwd<2>(a, cb, st); break;
            default: rc = launch_fwd<3>(a, cb, st); break;
        }
        if (rc) return rc;
    }
    return GS_OK;
}

extern "C" int gs_project_bwd(const gs_config* cfg, int64_t N, const float* means, const float* log_scales,
                              const float* quats, const float* opacity_logits, const float* sh, int32_t C,
                              const gs_camera* cams, const int32_t* radii, const float* dL_dmeans2d,
                              const float* dL_dconics, const float* dL_dopacities, const float* dL_drgbs,
                              float* dL_dmeans, float* dL_dlog_scales, float* dL_dquats, float* dL_dopacity_logits,
                              float* dL_dsh, int32_t accumulate, void* stream) {
    int rc = check_cfg(cfg);
    if (rc) return rc;
    rc = check_cams(C, cams);
    if (rc) return rc;
    if (N < 0) return GS_ERR_INVALID_ARGUMENT;
    if (N == 0) return GS_OK;
    if (!means || !log_scales || !quats || !opacity_logits || !sh || !radii || !dL_dmeans2d || !dL_dconics ||
        !dL_dopacities || !dL_drgbs || !dL_dmeans || !dL_dlog_scales || !dL_dquats || !dL_dopacity_logits || !dL_dsh)
        return GS_ERR_INVALID_ARGUMENT;
    if (!aligned(quats, 16) || !aligned(sh, 16) || !aligned(dL_dquats, 16) || !aligned(dL_dsh, 16) || !aligned(dL_dmeans2d, 8))
        return GS_ERR_INVALID_ARGUMENT;
    if ((N + kProjThreads - 1) / kProjThreads > 0x7fffffffLL || (int64_t)C * N >= (1LL << 31)) return GS_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    for (int c0 = 0; c0 < C; c0 += kMaxCamsPerLaunch) {
        const int nc = C - c0 < kMaxCamsPerLaunch ? C - c0 : kMaxCamsPerLaunch;
        CamBatch cb;
        for (int c = 0; c < nc; ++c) cb.cam[c] = make_devcam(cams[c0 + c]);
        ProjBwdArgs a;
        a.N = N; a.C = nc;
        a.means = means; a.log_scales = log_scales; a.quats = quats; a.logits = opacity_logits; a.sh = sh;
        const int64_t off = (int64_t)c0 * N;
        a.radii = radii + off;
        a.g_means2d = dL_dmeans2d + 2 * off; a.g_conics = dL_dconics + 3 * off;
        a.g_opacities = dL_dopacities + off; a.g_rgbs = dL_drgbs + 3 * off;
        a.d_means = dL_dmeans; a.d_log_scales = dL_dlog_scales; a.d_quats = dL_dquats;
        a.d_logits = dL_dopacity_logits; a.d_sh = dL_dsh;
        a.dilation = cfg->dilation;
        // the first chunk of cameras overwrites (unless the caller accumulates), later chunks add
        a.accumulate = (accumulate != 0 || c0 > 0) ? 1 : 0;
        switch (cfg->sh_degree) {
            case 0: rc = launch_bwd<0>(a, cb, st); break;
            case 1: rc = launch_bwd<1>(a, cb, st); break;
            case 2: rc = launch_bwd<2>(a, cb, st); break;
            default: rc = launch_bwd<3>(a, cb, st); break;
        }
        if (rc) return rc;
    }
    return GS_OK;
}
