// ssim.cu -- fused L1 + SSIM image loss, forward and backward (gs_l1_ssim_loss).
//
// L = (1 - lambda) mean|x - y| + lambda (1 - mean SSIM(x, y)) with the 11 x 11 Gaussian window (sigma 1.5), zero
// padding, C1 = 0.01^2, C2 = 0.03^2 ("computes the loss"; refs [31], [20]).  Two kernels over 16 x 16 pixel
// tiles of the [C, H, W, 3] images, both with the window applied separably out of shared memory:
//   ssim_stats_kernel   halo tiles (26 x 26 pixels, 3 interleaved channels) of x and y -> the five window means
//                       (x, y, x^2, y^2, xy) -> SSIM, its partial derivatives with respect to the three means that
//                       depend on x (pre-multiplied by -lambda / n) into three maps, and the loss sums;
//   ssim_grad_kernel    halo tiles of the three maps -> their window means (the adjoint of a symmetric, zero-padded
//                       correlation is the same correlation) -> dL/dx = g_mu + 2 x g_11 + y g_12 + L1 term.
// Algorithmic HBM bytes per pixel and channel: read x, y (8), write 3 maps (12); read 3 maps, x, y (20), write dL (4).
#include "common.cuh"

namespace gs {

constexpr int kSsimTile = 16;
constexpr int kSsimR = 5;
constexpr int kSsimWin = 2 * kSsimR + 1;
constexpr int kSsimHalo = kSsimTile + 2 * kSsimR;       // 26
constexpr int kSsimRow = kSsimHalo * 3;                 // floats per halo row (3 interleaved channels)
constexpr int kSsimRowPad = kSsimRow + 1;               // odd stride: column walks of the vertical pass spread over banks
constexpr float kSsimC1 = 0.01f * 0.01f;
constexpr float kSsimC2 = 0.03f * 0.03f;

struct SsimArgs {
    int32_t C, H, W;
    const float* x; const float* y;
    float* maps;            // [3][C, H, W, 3]: weighted dS/dmu1 (total), dS/ds11, dS/ds12
    float* dL; float* loss;
    int64_t n;              // C * H * W * 3
    float lambda, inv_n;
    float win[kSsimWin];
};

// rows i0-5 .. i0+20, pixels j0-5 .. j0+20 of view v, all three channels, zero outside the image
__device__ __forceinline__ void load_halo(const float* __restrict__ img, int v, int i0, int j0, int H, int W, float (*s)[kSsimRowPad]) {
    for (int k = threadIdx.x; k < kSsimHalo * kSsimRow; k += blockDim.x) {
        const int r = k / kSsimRow, c = k - r * kSsimRow;
        const int gi = i0 - kSsimR + r, gj = j0 - kSsimR + c / 3;
        float val = 0.0f;
        if (gi >= 0 && gi < H && gj >= 0 && gj < W) val = __ldg(img + ((int64_t)(v * (int64_t)H + gi) * W + (j0 - kSsimR)) * 3 + c);
        s[r][c] = val;
    }
}

__device__ __forceinline__ float block_sum(float v, float* s_red) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
    __syncthreads();
    float t = 0.0f;
    if (threadIdx.x == 0)
        for (int w = 0; w < 8; ++w) t += s_red[w];
    __syncthreads();
    return t;               // valid in thread 0
}

__global__ void __launch_bounds__(256) ssim_stats_kernel(const SsimArgs a) {
    __shared__ float sx[kSsimHalo][kSsimRowPad], sy[kSsimHalo][kSsimRowPad];
    __shared__ float hz[5][kSsimHalo][kSsimTile + 1];
    __shared__ float s_red[8];
    const int v = blockIdx.z, i0 = blockIdx.y * kSsimTile, j0 = blockIdx.x * kSsimTile;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    load_halo(a.x, v, i0, j0, a.H, a.W, sx);
    load_halo(a.y, v, i0, j0, a.H, a.W, sy);
    __syncthreads();
    const int gi = i0 + ty, gj = j0 + tx;
    const bool inside = gi < a.H && gj < a.W;
    const int64_t pix = ((int64_t)v * a.H + gi) * a.W + gj;
    const float wgt = -a.lambda * a.inv_n;
    float ssim_sum = 0.0f, l1_sum = 0.0f;
    for (int ch = 0; ch < 3; ++ch) {
        // horizontal pass: 26 rows x 16 columns, five quantities
        for (int k = threadIdx.x; k < kSsimHalo * kSsimTile; k += 256) {
            const int r = k >> 4, c = k & 15;
            float m1 = 0.f, m2 = 0.f, e11 = 0.f, e22 = 0.f, e12 = 0.f;
#pragma unroll
            for (int t = 0; t < kSsimWin; ++t) {
                const float w = a.win[t];
                const float xv = sx[r][(c + t) * 3 + ch], yv = sy[r][(c + t) * 3 + ch];
                m1 = fmaf(w, xv, m1); m2 = fmaf(w, yv, m2);
                e11 = fmaf(w * xv, xv, e11); e22 = fmaf(w * yv, yv, e22); e12 = fmaf(w * xv, yv, e12);
            }
            hz[0][r][c] = m1; hz[1][r][c] = m2; hz[2][r][c] = e11; hz[3][r][c] = e22; hz[4][r][c] = e12;
        }
        __syncthreads();
        // vertical pass at this thread's pixel
        float mu1 = 0.f, mu2 = 0.f, e11 = 0.f, e22 = 0.f, e12 = 0.f;
#pragma unroll
        for (int t = 0; t < kSsimWin; ++t) {
            const float w = a.win[t];
            mu1 = fmaf(w, hz[0][ty + t][tx], mu1); mu2 = fmaf(w, hz[1][ty + t][tx], mu2);
            e11 = fmaf(w, hz[2][ty + t][tx], e11); e22 = fmaf(w, hz[3][ty + t][tx], e22); e12 = fmaf(w, hz[4][ty + t][tx], e12);
        }
        if (inside) {
            const float s11 = e11 - mu1 * mu1, s22 = e22 - mu2 * mu2, s12 = e12 - mu1 * mu2;
            const float A1 = fmaf(2.0f * mu1, mu2, kSsimC1), A2 = fmaf(2.0f, s12, kSsimC2);
            const float B1 = fmaf(mu1, mu1, fmaf(mu2, mu2, kSsimC1)), B2 = s11 + s22 + kSsimC2;
            const float inv = 1.0f / (B1 * B2);
            const float S = A1 * A2 * inv;
            const float d11 = -S / B2;                                   // dS/ds11
            const float d12 = 2.0f * A1 * inv;                           // dS/ds12
            const float dmu = 2.0f * mu2 * A2 * inv - 2.0f * mu1 * S / B1 - 2.0f * mu1 * d11 - mu2 * d12;   // total dS/dmu1
            const int64_t o = 3 * pix + ch;
            a.maps[o] = wgt * dmu;
            a.maps[a.n + o] = wgt * d11;
            a.maps[2 * a.n + o] = wgt * d12;
            ssim_sum += S;
            l1_sum += fabsf(sx[ty + kSsimR][(tx + kSsimR) * 3 + ch] - sy[ty + kSsimR][(tx + kSsimR) * 3 + ch]);
        }
        __syncthreads();        // hz is rewritten for the next channel
    }
    const float part = (1.0f - a.lambda) * l1_sum * a.inv_n - a.lambda * ssim_sum * a.inv_n;
    float tot = block_sum(part, s_red);
    if (threadIdx.x == 0) {
        if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) tot += a.lambda;     // the constant of lambda (1 - mean SSIM)
        atomicAdd(a.loss, tot);
    }
}

__global__ void __launch_bounds__(256) ssim_grad_kernel(const SsimArgs a) {
    __shared__ float sm[3][kSsimHalo][kSsimRowPad];
    __shared__ float hz[3][kSsimHalo][kSsimTile + 1];
    const int v = blockIdx.z, i0 = blockIdx.y * kSsimTile, j0 = blockIdx.x * kSsimTile;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
#pragma unroll
    for (int q = 0; q < 3; ++q) load_halo(a.maps + q * a.n, v, i0, j0, a.H, a.W, sm[q]);
    __syncthreads();
    const int gi = i0 + ty, gj = j0 + tx;
    const bool inside = gi < a.H && gj < a.W;
    const int64_t pix = ((int64_t)v * a.H + gi) * a.W + gj;
    const float l1w = (1.0f - a.lambda) * a.inv_n;
    for (int ch = 0; ch < 3; ++ch) {
        for (int k = threadIdx.x; k < kSsimHalo * kSsimTile; k += 256) {
            const int r = k >> 4, c = k & 15;
            float g0 = 0.f, g1 = 0.f, g2 = 0.f;
#pragma unroll
            for (int t = 0; t < kSsimWin; ++t) {
                const float w = a.win[t];
                g0 = fmaf(w, sm[0][r][(c + t) * 3 + ch], g0);
                g1 = fmaf(w, sm[1][r][(c + t) * 3 + ch], g1);
                g2 = fmaf(w, sm[2][r][(c + t) * 3 + ch], g2);
            }
            hz[0][r][c] = g0; hz[1][r][c] = g1; hz[2][r][c] = g2;
        }
        __syncthreads();
        float g0 = 0.f, g1 = 0.f, g2 = 0.f;
#pragma unroll
        for (int t = 0; t < kSsimWin; ++t) {
            const float w = a.win[t];
            g0 = fmaf(w, hz[0][ty + t][tx], g0); g1 = fmaf(w, hz[1][ty + t][tx], g1); g2 = fmaf(w, hz[2][ty + t][tx], g2);
        }
        if (inside) {
            const int64_t o = 3 * pix + ch;
            const float xv = __ldg(a.x + o), yv = __ldg(a.y + o);
            const float d = xv - yv;
            const float l1 = d > 0.f ? l1w : (d < 0.f ? -l1w : 0.f);
            a.dL[o] = fmaf(2.0f * xv, g1, fmaf(yv, g2, g0)) + l1;
        }
        __syncthreads();
    }
}

}  // namespace gs

using namespace gs;

extern "C" int gs_l1_ssim_loss(int32_t C, int32_t height, int32_t width, const float* image, const float* target, float lambda,
                               float* dL_dimage, float* loss_sum, void* workspace, size_t* workspace_bytes, void* stream) {
    if (C < 1 || height < 1 || width < 1 || C > 65535 || height > 65536 || width > 65536) return GS_ERR_INVALID_ARGUMENT;
    if (!(lambda >= 0.0f) || !(lambda <= 1.0f)) return GS_ERR_INVALID_ARGUMENT;
    const int64_t n = (int64_t)C * height * width * 3;
    const size_t need = (size_t)3 * (size_t)n * sizeof(float);
    if (!workspace) {
        if (!workspace_bytes) return GS_ERR_INVALID_ARGUMENT;
        *workspace_bytes = need;
        return GS_OK;
    }
    if (workspace_bytes && *workspace_bytes < need) return GS_ERR_INVALID_ARGUMENT;
    if (!image || !target || !dL_dimage || !loss_sum || !aligned(workspace, 4)) return GS_ERR_INVALID_ARGUMENT;
    SsimArgs a;
    a.C = C; a.H = height; a.W = width;
    a.x = image; a.y = target; a.maps = reinterpret_cast<float*>(workspace); a.dL = dL_dimage; a.loss = loss_sum;
    a.n = n; a.lambda = lambda; a.inv_n = (float)(1.0 / (double)n);
    // window: exp(-k^2 / (2 sigma^2)), sigma = 1.5, normalised in double, rounded once
    double g[kSsimWin], sum = 0.0;
    for (int k = 0; k < kSsimWin; ++k) {
        const double d = (double)(k - kSsimR);
        g[k] = exp(-d * d / (2.0 * 1.5 * 1.5));
        sum += g[k];
    }
    for (int k = 0; k < kSsimWin; ++k) a.win[k] = (float)(g[k] / sum);
    const dim3 grid((unsigned)((width + kSsimTile - 1) / kSsimTile), (unsigned)((height + kSsimTile - 1) / kSsimTile), (unsigned)C);
    cudaStream_t st = (cudaStream_t)stream;
    ssim_stats_kernel<<<grid, 256, 0, st>>>(a);
    int rc = launch_status();
    if (rc) return rc;
    ssim_grad_kernel<<<grid, 256, 0, st>>>(a);
    return launch_status();
}
