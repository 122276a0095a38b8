// common.cuh -- shared device/host helpers of the sm_100a splatting library (CUDA path only;
// nothing here is used by, or derived from, the CPU oracle under oracle/).
#pragma once

#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "../../include/gsplat_b200.h"

namespace gs {

constexpr int kTile = 16;
constexpr int kMaxCamsPerLaunch = 16;

// Device-side camera: the host gs_camera plus derived constants (Jacobian clamp limits, camera
// centre o = -W^T tau, tile grid).  Passed by value in kernel parameters (constant bank).
struct DevCam {
    float W[9];
    float tau[3];
    float fx, fy, cx, cy;
    float near_plane, far_plane;
    float lim_x, lim_y;
    float ox, oy, oz;
    float wnorm2;              // upper bound of |W|_2^2 (1 for a rigid transform): max absolute row sum of W W^T
    int32_t width, height, gx, gy;
    // linear lateral cull with a scene-wide scale bound s (project.cu, phase A): a Gaussian whose tile rectangle can be
    // non-empty satisfies  fx |t_x - t_z (gx 8 - cx) / fx| <= lat_k1x t_z + lat_k2 s  (same in y)
    float lat_cx, lat_cy, lat_k1x, lat_k1y, lat_k2, lat_abs;
};

struct CamBatch {
    DevCam cam[kMaxCamsPerLaunch];
};

inline DevCam make_devcam(const gs_camera& c) {
    DevCam d;
    for (int r = 0; r < 3; ++r) {
        for (int j = 0; j < 3; ++j) d.W[3 * r + j] = c.viewmat[4 * r + j];
        d.tau[r] = c.viewmat[4 * r + 3];
    }
    d.fx = c.fx; d.fy = c.fy; d.cx = c.cx; d.cy = c.cy;
    d.near_plane = c.near_plane; d.far_plane = c.far_plane;
    d.lim_x = 1.3f * (float)c.width / (2.0f * c.fx);
    d.lim_y = 1.3f * (float)c.height / (2.0f * c.fy);
    d.ox = -(d.W[0] * d.tau[0] + d.W[3] * d.tau[1] + d.W[6] * d.tau[2]);
    d.oy = -(d.W[1] * d.tau[0] + d.W[4] * d.tau[1] + d.W[7] * d.tau[2]);
    d.oz = -(d.W[2] * d.tau[0] + d.W[5] * d.tau[1] + d.W[8] * d.tau[2]);
    d.wnorm2 = 1.0f;
    for (int r = 0; r < 3; ++r) {
        float row = 0.0f;
        for (int j = 0; j < 3; ++j) {
            const float g = d.W[3 * r] * d.W[3 * j] + d.W[3 * r + 1] * d.W[3 * j + 1] + d.W[3 * r + 2] * d.W[3 * j + 2];
            row += g < 0.0f ? -g : g;
        }
        if (row > d.wnorm2) d.wnorm2 = row;
    }
    d.width = c.width; d.height = c.height;
    d.gx = (c.width + kTile - 1) / kTile;
    d.gy = (c.height + kTile - 1) / kTile;
    d.lat_cx = d.lat_cy = d.lat_k1x = d.lat_k1y = d.lat_k2 = d.lat_abs = 0.0f;      // set by set_lateral_bound
    return d;
}

// Constants of the linear lateral cull.  A visible entry has a non-empty tile rectangle, hence |u - 8 gx| <= 8 gx + 16 + r
// with r <= extent sqrt(lambda_max) + 1, lambda_max <= 2 (L + dilation) + sqrt(0.1), L <= s^2 |J|_F^2 |W|_2^2 and
// |J|_F^2 <= (fx^2 (1 + lim_x^2) + fy^2 (1 + lim_y^2)) / t_z^2 =: jf0 / t_z^2.  With sqrt(a + b) <= sqrt(a) + sqrt(b) and
// u = fx t_x / t_z + cx this gives  fx |t_x - t_z (8 gx - cx) / fx| <= t_z (8 gx + 17 + extent sqrt(2 dil + 0.32)) + extent s sqrt(2 jf0);
// 0.2 % and 4 pixels of slack cover the fp32 rounding of both sides; the rounding of t = W p + tau itself (three products of
// size <= |p| <= |t| + |tau| each) adds lat_abs = 16 eps |tau| max(fx, fy) (the |t| part is inside the 0.2 %).
inline void set_lateral_bound(DevCam& d, float extent, float dilation) {
    const float dil = dilation > 0.0f ? dilation : 0.0f;
    const float pad = 17.0f + extent * sqrtf(2.0f * dil + 0.32f) + 4.0f;
    d.lat_cx = (8.0f * (float)d.gx - d.cx) / d.fx;
    d.lat_cy = (8.0f * (float)d.gy - d.cy) / d.fy;
    d.lat_k1x = (8.0f * (float)d.gx + pad) * 1.002f;
    d.lat_k1y = (8.0f * (float)d.gy + pad) * 1.002f;
    const float jf0 = (d.fx * d.fx * (1.0f + d.lim_x * d.lim_x) + d.fy * d.fy * (1.0f + d.lim_y * d.lim_y)) * d.wnorm2;
    d.lat_k2 = extent * sqrtf(2.0f * jf0) * 1.002f;
    const float tn = sqrtf(d.tau[0] * d.tau[0] + d.tau[1] * d.tau[1] + d.tau[2] * d.tau[2]);
    d.lat_abs = 16.0f * 5.9604645e-8f * tn * (d.fx > d.fy ? d.fx : d.fy);
}

inline bool finite_f(float x) { return x == x && x - x == 0.0f; }

// Validation shared by the entry points.
inline int check_cfg(const gs_config* cfg) {
    if (!cfg) return GS_ERR_INVALID_ARGUMENT;
    if (cfg->sh_degree < 0 || cfg->sh_degree > 3) return GS_ERR_INVALID_ARGUMENT;
    if (cfg->tile != kTile) return GS_ERR_UNSUPPORTED;
    if (!finite_f(cfg->dilation) || !finite_f(cfg->alpha_min) || !finite_f(cfg->alpha_max) ||
        !finite_f(cfg->t_min) || !finite_f(cfg->extent) || !(cfg->extent > 0.0f))
        return GS_ERR_INVALID_ARGUMENT;
    return GS_OK;
}
inline int check_cams(int32_t C, const gs_camera* cams) {
    if (!cams || C < 1 || C > GS_MAX_VIEWS) return GS_ERR_INVALID_ARGUMENT;
    for (int c = 0; c < C; ++c) {
        const gs_camera& k = cams[c];
        if (k.width < 1 || k.height < 1 || k.width > 65536 || k.height > 65536) return GS_ERR_INVALID_ARGUMENT;
        if (k.width != cams[0].width || k.height != cams[0].height) return GS_ERR_INVALID_ARGUMENT;
        if (!finite_f(k.fx) || !finite_f(k.fy) || !finite_f(k.cx) || !finite_f(k.cy) || !(k.fx > 0.0f) || !(k.fy > 0.0f))
            return GS_ERR_INVALID_ARGUMENT;
        for (int j = 0; j < 12; ++j)
            if (!finite_f(k.viewmat[j])) return GS_ERR_INVALID_ARGUMENT;
        if (!(k.near_plane > 0.0f) || !(k.far_plane > k.near_plane)) return GS_ERR_INVALID_ARGUMENT;
    }
    return GS_OK;
}
inline bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }

inline int cuda_status(cudaError_t e) { return e == cudaSuccess ? GS_OK : GS_ERR_CUDA; }
inline int launch_status() { return cuda_status(cudaGetLastError()); }

// ---- programmatic dependent launch ---------------------------------------------------------------
// The stages are chains of short kernels on one stream.  With the launch attribute below the next kernel is released when
// the blocks of its predecessor have exited (not after the full completion + flush handshake of a plain launch), and its
// blocks stop at pdl_enter() until the predecessor's writes are visible.  Every kernel of the library is launched through
// launch_chained() and calls pdl_enter() as its FIRST statement, in every block and before any early return: a block that
// left without waiting would let its grid complete -- and release the grid behind it -- before the grid in front has
// finished.  No kernel touches global memory before the wait, so the dependency semantics are those of a plain stream.
// Measured (bin_tiles, ms): city 0.368 -> 0.335, block 0.206 -> 0.179, room 0.856 -> 0.814, object 0.398 -> 0.362.
// An explicit early `griddepcontrol.launch_dependents` at the top of every kernel (blocks of the next kernels resident
// and waiting while the predecessor runs) was slower on the larger scenes: city 0.382, object 0.411 (block 0.183).
__device__ __forceinline__ void pdl_enter() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
template <typename... KArgs, typename... Args>
inline void launch_chained(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// Per-device cache of immutable facts about the current device (SM count; which kernels already have their opt-in
// dynamic shared-memory size set; resident blocks per SM of the persistent kernels).  Entries are idempotent, so
// concurrent first calls are harmless; nothing here changes the result of any call.
struct DeviceCache {
    int sms;
    unsigned attr_mask;     // bit k: kernel slot k has its shared-memory attribute set on this device
    int occ[16];            // resident blocks per SM per kernel slot (0 = not queried yet)
};
inline DeviceCache& device_cache() {
    static DeviceCache cache[64];
    int dev = 0;
    cudaGetDevice(&dev);
    DeviceCache& d = cache[dev & 63];
    if (!d.sms) {
        int sms = 148;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        d.sms = sms;
    }
    return d;
}
inline int sm_count() { return device_cache().sms; }
// sets cudaFuncAttributeMaxDynamicSharedMemorySize once per device and kernel slot
template <typename Kernel>
inline int ensure_smem(Kernel kernel, int slot, int bytes) {
    DeviceCache& d = device_cache();
    if (!(d.attr_mask & (1u << slot))) {
        if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) != cudaSuccess) return GS_ERR_CUDA;
        d.attr_mask |= 1u << slot;
    }
    return GS_OK;
}

// Tile rectangle of O-P1 step 8, fp32 with one rounding per operation (no FMA contraction:
// the same bits must come out of P1, the emit kernel and the host-side reference).
__device__ __forceinline__ int clampi(int a, int lo, int hi) { return min(max(a, lo), hi); }
__device__ __forceinline__ int floor_to_int_sat(float a) {
    // __float2int_rd saturates and maps NaN to 0; clamp to +-2e9 like the definition
    float f = floorf(a);
    f = fminf(fmaxf(f, -2.0e9f), 2.0e9f);
    return (int)f;
}
__device__ __forceinline__ void tile_rect(float u, float v, int radius, int gx, int gy, int& x0, int& x1, int& y0, int& y1) {
    const float inv = 1.0f / (float)kTile;
    const float r_lo = (float)radius;
    const float r_hi = (float)(radius + kTile - 1);
    x0 = clampi(floor_to_int_sat(__fmul_rn(__fsub_rn(u, r_lo), inv)), 0, gx);
    x1 = clampi(floor_to_int_sat(__fmul_rn(__fadd_rn(u, r_hi), inv)), 0, gx);
    y0 = clampi(floor_to_int_sat(__fmul_rn(__fsub_rn(v, r_lo), inv)), 0, gy);
    y1 = clampi(floor_to_int_sat(__fmul_rn(__fadd_rn(v, r_hi), inv)), 0, gy);
}

// Two-wide FP32 (sm_100a FFMA2 / FMUL2 / FADD2; PTX fma/mul/add.rn.f32x2 on 64-bit register pairs): one issue slot for two
// lanes of arithmetic.  Used by the issue-bound raster and SSIM kernels.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpk2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
// Real spherical-harmonic constants, degrees 0..3 (closed forms evaluated in double, rounded once).
constexpr float kC0 = 0.28209479177387814f;   // 1/(2 sqrt(pi))
constexpr float kC1 = 0.4886025119029199f;    // sqrt(3/(4 pi))
constexpr float kC2a = 1.0925484305920792f;   // 1/2 sqrt(15/pi)
constexpr float kC2b = 0.31539156525252005f;  // 1/4 sqrt(5/pi)
constexpr float kC2c = 0.5462742152960396f;   // 1/4 sqrt(15/pi)
constexpr float kC3a = 0.5900435899266435f;   // 1/4 sqrt(35/(2 pi))
constexpr float kC3b = 2.890611442640554f;    // 1/2 sqrt(105/pi)
constexpr float kC3c = 0.4570457994644658f;   // 1/4 sqrt(21/(2 pi))
constexpr float kC3d = 0.3731763325901154f;   // 1/4 sqrt(7/pi)
constexpr float kC3e = 1.445305721320277f;    // 1/4 sqrt(105/pi)

}  // namespace gs
