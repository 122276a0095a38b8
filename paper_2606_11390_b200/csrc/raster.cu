// raster.cu -- per-pixel stages R1 (gs_raster_fwd) and R2 (gs_raster_bwd) plus the harness L1 loss.
//
// One 16x16 thread block per (view, tile).  The tile's sorted records are staged through shared
// memory in batches of 256 (one gathered record per thread), every thread then walks the batch for
// its pixel.  Forward: a warp leaves the batch loop as soon as all of its 32 pixels are saturated and
// the block stops fetching when every warp has.  Backward: back-to-front from
// the tile's largest n_contrib, per-record partial sums are reduced inside the warp with a
// value-splitting butterfly (14 shuffles for 9 values), combined across the block's warps in shared
// memory and flushed with one device-scope atomic per value and record.
#include "common.cuh"

namespace gs {

constexpr int kBlock = kTile * kTile;  // 256

struct RasterArgs {
    int32_t width, height, gx, gy;
    int64_t tiles;
    const int32_t* vals; const int64_t* ranges;
    const float* means2d; const float* conics; const float* opacities; const float* rgbs;
    float bg0, bg1, bg2;
    float alpha_min, alpha_max, t_min;
};

struct RasterFwdOut {
    float* image; float* final_T; int32_t* n_contrib;
};

__global__ void __launch_bounds__(kBlock) raster_fwd_kernel(const RasterArgs a, const RasterFwdOut o) {
    __shared__ float4 s_geo[kBlock];   // u, v, A, B
    __shared__ float4 s_col[kBlock];   // C, opacity, r, g
    __shared__ float s_b[kBlock];      // b
    const int tid = threadIdx.x;
    const int64_t bt = blockIdx.x;                  // view * tiles + tile
    const int64_t view = bt / a.tiles;
    const int t = (int)(bt - view * a.tiles);
    const int ty = t / a.gx, tx = t - ty * a.gx;
    const int j = tx * kTile + (tid & (kTile - 1));
    const int i = ty * kTile + (tid >> 4);
    const bool inside = (i < a.height) && (j < a.width);
    const float px = (float)j + 0.5f, py = (float)i + 0.5f;

    const int64_t start = __ldg(a.ranges + 2 * bt), end = __ldg(a.ranges + 2 * bt + 1);
    float T = 1.0f, c0 = 0.f, c1 = 0.f, c2 = 0.f;
    int last = 0;
    bool done = !inside;
    for (int64_t base = start; base < end; base += kBlock) {
        if (__syncthreads_and(done)) break;
        const int64_t k = base + tid;
        if (k < end) {
            const int g = __ldg(a.vals + k);
            const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + g);
            const float A = __ldg(a.conics + 3 * (int64_t)g), B = __ldg(a.conics + 3 * (int64_t)g + 1), Cc = __ldg(a.conics + 3 * (int64_t)g + 2);
            s_geo[tid] = make_float4(uv.x, uv.y, A, B);
            s_col[tid] = make_float4(Cc, __ldg(a.opacities + g), __ldg(a.rgbs + 3 * (int64_t)g), __ldg(a.rgbs + 3 * (int64_t)g + 1));
            s_b[tid] = __ldg(a.rgbs + 3 * (int64_t)g + 2);
        }
        __syncthreads();
        const int cnt = (int)((end - base) < kBlock ? (end - base) : kBlock);
        const int nbase = (int)(base - start);
        for (int q = 0; q < cnt && !done; ++q) {
            const float4 ge = s_geo[q];
            const float4 co = s_col[q];
            const float dx = ge.x - px, dy = ge.y - py;
            const float power = -0.5f * (ge.z * dx * dx + co.x * dy * dy) - ge.w * dx * dy;
            if (power > 0.0f) continue;
            const float alpha = fminf(a.alpha_max, co.y * __expf(power));
            if (alpha < a.alpha_min) continue;
            const float Tn = T * (1.0f - alpha);
            if (Tn < a.t_min) { done = true; break; }
            const float wgt = alpha * T;
            c0 = fmaf(co.z, wgt, c0);
            c1 = fmaf(co.w, wgt, c1);
            c2 = fmaf(s_b[q], wgt, c2);
            T = Tn;
            last = nbase + q + 1;
        }
    }
    if (inside) {
        const int64_t pix = (view * a.height + i) * a.width + j;
        o.image[3 * pix] = c0 + T * a.bg0;
        o.image[3 * pix + 1] = c1 + T * a.bg1;
        o.image[3 * pix + 2] = c2 + T * a.bg2;
        o.final_T[pix] = T;
        o.n_contrib[pix] = last;
    }
}

// ---------------------------------------------------------------------------------------------
struct RasterBwdIO {
    const float* final_T; const int32_t* n_contrib; const float* dL_dimage;
    float* g_means2d; float* g_conics; float* g_opacities; float* g_rgbs;
};

// Reduce 9 per-lane values over the warp.  Values 0..7 use a splitting butterfly (each exchange
// halves the number of values a lane carries): 4 + 2 + 1 + 1 + 1 shuffles; value 8 takes the plain
// 5-step butterfly.  On return lane (4*k) holds the warp total of value k (k = 0..7, bit pattern
// k = lane bits 4..2) in `out8`, and every lane holds the total of value 8 in `out9`.
__device__ __forceinline__ void warp_reduce9(const float v[9], int lane, float& out8, float& out9) {
    const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
    float a0, a1, a2, a3;
    {
        const float s0 = b4 ? v[0] : v[4], s1 = b4 ? v[1] : v[5], s2 = b4 ? v[2] : v[6], s3 = b4 ? v[3] : v[7];
        const float k0 = b4 ? v[4] : v[0], k1 = b4 ? v[5] : v[1], k2 = b4 ? v[6] : v[2], k3 = b4 ? v[7] : v[3];
        a0 = k0 + __shfl_xor_sync(0xffffffffu, s0, 16);
        a1 = k1 + __shfl_xor_sync(0xffffffffu, s1, 16);
        a2 = k2 + __shfl_xor_sync(0xffffffffu, s2, 16);
        a3 = k3 + __shfl_xor_sync(0xffffffffu, s3, 16);
    }
    float c0, c1;
    {
        const float s0 = b3 ? a0 : a2, s1 = b3 ? a1 : a3;
        const float k0 = b3 ? a2 : a0, k1 = b3 ? a3 : a1;
        c0 = k0 + __shfl_xor_sync(0xffffffffu, s0, 8);
        c1 = k1 + __shfl_xor_sync(0xffffffffu, s1, 8);
    }
    float e;
    {
        const float s = b2 ? c0 : c1;
        const float k = b2 ? c1 : c0;
        e = k + __shfl_xor_sync(0xffffffffu, s, 4);
    }
    e += __shfl_xor_sync(0xffffffffu, e, 2);
    e += __shfl_xor_sync(0xffffffffu, e, 1);
    out8 = e;
    float w = v[8];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) w += __shfl_xor_sync(0xffffffffu, w, d);
    out9 = w;
}

__global__ void __launch_bounds__(kBlock) raster_bwd_kernel(const RasterArgs a, const RasterBwdIO io) {
    __shared__ float4 s_geo[kBlock];   // u, v, A, B
    __shared__ float4 s_col[kBlock];   // C, opacity, r, g
    __shared__ float s_b[kBlock];
    __shared__ int s_id[kBlock];
    __shared__ float s_acc[kBlock][9]; // per record: du, dv, dA, dB, dC, do, dr, dg | db
    __shared__ int s_max;
    const int tid = threadIdx.x, lane = tid & 31;
    const int64_t bt = blockIdx.x;
    const int64_t view = bt / a.tiles;
    const int t = (int)(bt - view * a.tiles);
    const int ty = t / a.gx, tx = t - ty * a.gx;
    const int j = tx * kTile + (tid & (kTile - 1));
    const int i = ty * kTile + (tid >> 4);
    const bool inside = (i < a.height) && (j < a.width);
    const float px = (float)j + 0.5f, py = (float)i + 0.5f;
    const int64_t start = __ldg(a.ranges + 2 * bt);

    float T = 0.f, g0 = 0.f, g1 = 0.f, g2 = 0.f;
    int ncon = 0;
    if (inside) {
        const int64_t pix = (view * a.height + i) * a.width + j;
        T = __ldg(io.final_T + pix);
        ncon = __ldg(io.n_contrib + pix);
        g0 = __ldg(io.dL_dimage + 3 * pix); g1 = __ldg(io.dL_dimage + 3 * pix + 1); g2 = __ldg(io.dL_dimage + 3 * pix + 2);
    }
    if (tid == 0) s_max = 0;
    __syncthreads();
    {
        int m = ncon;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, d));
        if (lane == 0 && m > 0) atomicMax(&s_max, m);
    }
    __syncthreads();
    const int maxn = s_max;
    if (maxn == 0) return;
    // colour accumulated behind the current record
    float S0 = a.bg0, S1 = a.bg1, S2 = a.bg2;
    const int nb = (maxn + kBlock - 1) / kBlock;
    for (int b = nb - 1; b >= 0; --b) {
        const int cnt = min(kBlock, maxn - b * kBlock);
        __syncthreads();   // previous batch fully flushed
        if (tid < cnt) {
            const int g = __ldg(a.vals + start + (int64_t)b * kBlock + tid);
            const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + g);
            const float A = __ldg(a.conics + 3 * (int64_t)g), B = __ldg(a.conics + 3 * (int64_t)g + 1), Cc = __ldg(a.conics + 3 * (int64_t)g + 2);
            s_geo[tid] = make_float4(uv.x, uv.y, A, B);
            s_col[tid] = make_float4(Cc, __ldg(a.opacities + g), __ldg(a.rgbs + 3 * (int64_t)g), __ldg(a.rgbs + 3 * (int64_t)g + 1));
            s_b[tid] = __ldg(a.rgbs + 3 * (int64_t)g + 2);
            s_id[tid] = g;
        }
#pragma unroll
        for (int k = 0; k < 9; ++k) s_acc[tid][k] = 0.f;
        __syncthreads();
        for (int q = cnt - 1; q >= 0; --q) {
            const int idx = b * kBlock + q;           // position of the record in the tile's list
            bool valid = idx < ncon;
            float v[9];
#pragma unroll
            for (int k = 0; k < 9; ++k) v[k] = 0.f;
            if (valid) {
                const float4 ge = s_geo[q];
                const float4 co = s_col[q];
                const float dx = ge.x - px, dy = ge.y - py;
                const float power = -0.5f * (ge.z * dx * dx + co.x * dy * dy) - ge.w * dx * dy;
                const float G = __expf(power);
                const float raw = co.y * G;
                const float alpha = fminf(a.alpha_max, raw);
                valid = (power <= 0.0f) && (alpha >= a.alpha_min);
                if (valid) {
                    const float cb = s_b[q];
                    T = T / (1.0f - alpha);          // transmittance in front of this record
                    const float wgt = alpha * T;
                    v[6] = wgt * g0; v[7] = wgt * g1; v[8] = wgt * g2;
                    const float dL_dalpha = T * ((co.z - S0) * g0 + (co.w - S1) * g1 + (cb - S2) * g2);
                    S0 = alpha * co.z + (1.0f - alpha) * S0;
                    S1 = alpha * co.w + (1.0f - alpha) * S1;
                    S2 = alpha * cb + (1.0f - alpha) * S2;
                    if (!(raw > a.alpha_max)) {       // no gradient through the alpha_max clamp
                        v[5] = G * dL_dalpha;
                        const float gp = alpha * dL_dalpha;
                        v[2] = -0.5f * dx * dx * gp;
                        v[3] = -dx * dy * gp;
                        v[4] = -0.5f * dy * dy * gp;
                        v[0] = -(ge.z * dx + ge.w * dy) * gp;
                        v[1] = -(ge.w * dx + co.x * dy) * gp;
                    }
                }
            }
            if (__any_sync(0xffffffffu, valid)) {
                float r8, r9;
                warp_reduce9(v, lane, r8, r9);
                if ((lane & 3) == 0) atomicAdd(&s_acc[q][lane >> 2], r8);
                if (lane == 1) atomicAdd(&s_acc[q][8], r9);
            }
        }
        __syncthreads();
        if (tid < cnt) {
            const int64_t g = s_id[tid];
            const float* acc = s_acc[tid];
            if (acc[0] != 0.f) atomicAdd(io.g_means2d + 2 * g, acc[0]);
            if (acc[1] != 0.f) atomicAdd(io.g_means2d + 2 * g + 1, acc[1]);
            if (acc[2] != 0.f) atomicAdd(io.g_conics + 3 * g, acc[2]);
            if (acc[3] != 0.f) atomicAdd(io.g_conics + 3 * g + 1, acc[3]);
            if (acc[4] != 0.f) atomicAdd(io.g_conics + 3 * g + 2, acc[4]);
            if (acc[5] != 0.f) atomicAdd(io.g_opacities + g, acc[5]);
            if (acc[6] != 0.f) atomicAdd(io.g_rgbs + 3 * g, acc[6]);
            if (acc[7] != 0.f) atomicAdd(io.g_rgbs + 3 * g + 1, acc[7]);
            if (acc[8] != 0.f) atomicAdd(io.g_rgbs + 3 * g + 2, acc[8]);
        }
    }
}

// zero the gradient rows of visible entries only (dense zero-fill when radii == nullptr is a memset)
__global__ void __launch_bounds__(256) zero_visible_rows_kernel(int64_t n, const int32_t* __restrict__ radii, float* g_means2d,
                                                                float* g_conics, float* g_opacities, float* g_rgbs) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    if (__ldg(radii + e) <= 0) return;
    reinterpret_cast<float2*>(g_means2d)[e] = make_float2(0.f, 0.f);
    g_conics[3 * e] = 0.f; g_conics[3 * e + 1] = 0.f; g_conics[3 * e + 2] = 0.f;
    g_opacities[e] = 0.f;
    g_rgbs[3 * e] = 0.f; g_rgbs[3 * e + 1] = 0.f; g_rgbs[3 * e + 2] = 0.f;
}

__global__ void __launch_bounds__(256) l1_loss_kernel(int64_t n, const float* __restrict__ image, const float* __restrict__ target,
                                                      float* __restrict__ dL, float* loss_sum, float inv_n) {
    float acc = 0.f;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        const float d = __ldg(image + k) - __ldg(target + k);
        acc += fabsf(d);
        dL[k] = d > 0.f ? inv_n : (d < 0.f ? -inv_n : 0.f);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    __shared__ float s[8];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        float tot = 0.f;
        for (int w = 0; w < 8; ++w) tot += s[w];
        atomicAdd(loss_sum, tot * inv_n);
    }
}

static int fill_args(const gs_config* cfg, int32_t C, const gs_camera* cams, const int32_t* vals, const int64_t* ranges,
                     const float* means2d, const float* conics, const float* opacities, const float* rgbs, const float* bg,
                     RasterArgs& a) {
    int rc = check_cfg(cfg);
    if (rc) return rc;
    rc = check_cams(C, cams);
    if (rc) return rc;
    if (!ranges || !means2d || !conics || !opacities || !rgbs || !bg || !aligned(means2d, 8)) return GS_ERR_INVALID_ARGUMENT;
    a.width = cams[0].width; a.height = cams[0].height;
    a.gx = (a.width + kTile - 1) / kTile; a.gy = (a.height + kTile - 1) / kTile;
    a.tiles = (int64_t)a.gx * a.gy;
    if ((int64_t)C * a.tiles > 0x7fffffffLL) return GS_ERR_UNSUPPORTED;
    a.vals = vals; a.ranges = ranges; a.means2d = means2d; a.conics = conics; a.opacities = opacities; a.rgbs = rgbs;
    a.bg0 = bg[0]; a.bg1 = bg[1]; a.bg2 = bg[2];
    a.alpha_min = cfg->alpha_min; a.alpha_max = cfg->alpha_max; a.t_min = cfg->t_min;
    return GS_OK;
}

}  // namespace gs

using namespace gs;

extern "C" int gs_raster_fwd(const gs_config* cfg, int32_t C, const gs_camera* cams, const int32_t* isect_vals,
                             const int64_t* tile_ranges, const float* means2d, const float* conics, const float* opacities,
                             const float* rgbs, const float* bg, float* image, float* final_T, int32_t* n_contrib, void* stream) {
    RasterArgs a;
    int rc = fill_args(cfg, C, cams, isect_vals, tile_ranges, means2d, conics, opacities, rgbs, bg, a);
    if (rc) return rc;
    if (!image || !final_T || !n_contrib) return GS_ERR_INVALID_ARGUMENT;
    RasterFwdOut o{image, final_T, n_contrib};
    raster_fwd_kernel<<<(unsigned)(C * a.tiles), kBlock, 0, (cudaStream_t)stream>>>(a, o);
    return launch_status();
}

extern "C" int gs_raster_bwd(const gs_config* cfg, int32_t C, const gs_camera* cams, int64_t N_total,
                             const int32_t* isect_vals, const int64_t* tile_ranges, const float* means2d, const float* conics,
                             const float* opacities, const float* rgbs, const float* bg, const float* final_T,
                             const int32_t* n_contrib, const float* dL_dimage, const int32_t* radii, float* dL_dmeans2d,
                             float* dL_dconics, float* dL_dopacities, float* dL_drgbs, void* stream) {
    RasterArgs a;
    int rc = fill_args(cfg, C, cams, isect_vals, tile_ranges, means2d, conics, opacities, rgbs, bg, a);
    if (rc) return rc;
    if (N_total < 0 || N_total >= (1LL << 31)) return GS_ERR_INVALID_ARGUMENT;
    if (!final_T || !n_contrib || !dL_dimage || !dL_dmeans2d || !dL_dconics || !dL_dopacities || !dL_drgbs || !aligned(dL_dmeans2d, 8))
        return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t st = (cudaStream_t)stream;
    if (N_total > 0) {
        if (radii) {
            zero_visible_rows_kernel<<<(unsigned)((N_total + 255) / 256), 256, 0, st>>>(N_total, radii, dL_dmeans2d, dL_dconics,
                                                                                         dL_dopacities, dL_drgbs);
            rc = launch_status();
            if (rc) return rc;
        } else {
            if (cudaMemsetAsync(dL_dmeans2d, 0, (size_t)N_total * 2 * sizeof(float), st) != cudaSuccess ||
                cudaMemsetAsync(dL_dconics, 0, (size_t)N_total * 3 * sizeof(float), st) != cudaSuccess ||
                cudaMemsetAsync(dL_dopacities, 0, (size_t)N_total * sizeof(float), st) != cudaSuccess ||
                cudaMemsetAsync(dL_drgbs, 0, (size_t)N_total * 3 * sizeof(float), st) != cudaSuccess)
                return GS_ERR_CUDA;
        }
    }
    RasterBwdIO io{final_T, n_contrib, dL_dimage, dL_dmeans2d, dL_dconics, dL_dopacities, dL_drgbs};
    raster_bwd_kernel<<<(unsigned)(C * a.tiles), kBlock, 0, st>>>(a, io);
    return launch_status();
}

extern "C" int gs_l1_loss(int64_t n, const float* image, const float* target, float* dL_dimage, float* loss_sum, void* stream) {
    if (n < 0) return GS_ERR_INVALID_ARGUMENT;
    if (n == 0) return GS_OK;
    if (!image || !target || !dL_dimage || !loss_sum) return GS_ERR_INVALID_ARGUMENT;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    int64_t blocks = (n + 255) / 256;
    if (blocks > (int64_t)sms * 16) blocks = (int64_t)sms * 16;
    l1_loss_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(n, image, target, dL_dimage, loss_sum, 1.0f / (float)n);
    return launch_status();
}

extern "C" int gs_config_default(gs_config* cfg) {
    if (!cfg) return GS_ERR_INVALID_ARGUMENT;
    cfg->dilation = 0.3f; cfg->alpha_min = 1.0f / 255.0f; cfg->alpha_max = 0.99f; cfg->t_min = 1.0e-4f; cfg->extent = 3.0f;
    cfg->tile = 16; cfg->sh_degree = 3;
    return GS_OK;
}

extern "C" const char* gs_status_string(int status) {
    switch (status) {
        case GS_OK: return "ok";
        case GS_ERR_INVALID_ARGUMENT: return "invalid argument";
        case GS_ERR_CAPACITY: return "intersection capacity too small";
        case GS_ERR_CUDA: return "CUDA error";
        case GS_ERR_UNSUPPORTED: return "unsupported size or configuration";
        default: return "unknown status";
    }
}
