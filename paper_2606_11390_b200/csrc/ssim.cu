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
#include <cuda.h>      // CUtensorMap (types only: the encoder is looked up at run time, the library does not link libcuda)

#include "common.cuh"

namespace gs {

constexpr int kSsimTile = 16;
constexpr int kSsimR = 5;
constexpr int kSsimWin = 2 * kSsimR + 1;
constexpr int kSsimHalo = kSsimTile + 2 * kSsimR;       // 26
constexpr int kSsimRow = kSsimHalo * 3;                 // floats per halo row (3 interleaved channels)
constexpr int kSsimRowPad = kSsimRow + 1;               // odd stride: column walks of the vertical pass spread over banks
constexpr int kSsimRowTma = 80;                         // TMA halo rows: 80 floats = 320 bytes (the box width must be a multiple of 16 bytes)
constexpr int kSsimTmaOff = 1;                          // ... starting one float left of the halo: the innermost start coordinate must be a
                                                        // multiple of 16 bytes (measured on B200: illegal instruction otherwise), and
                                                        // 3 (16 bx - 5) - 1 = 48 bx - 16 is
constexpr unsigned kSsimTmaBytes = kSsimHalo * kSsimRowTma * 4;
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

// rows i0-5 .. i0+20, pixels j0-5 .. j0+20 of view v, all three channels, zero outside the image; a warp takes whole
// rows (78 contiguous floats: three coalesced requests).  The elements go global -> shared with cp.async (4 bytes each,
// zero-filled outside the image), so every load of every halo tile of a block is in flight before the first wait.
template <int ROW>
__device__ __forceinline__ void load_halo_async(const float* __restrict__ img, int v, int i0, int j0, int H, int W, float (*s)[ROW]) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // per-thread column state (the same for every row): three elements c = lane + 32 it of the 78-float row
    bool col_in[3];
#pragma unroll
    for (int it = 0; it < 3; ++it) {
        const int c = lane + 32 * it;
        const int gj = j0 - kSsimR + c / 3;
        col_in[it] = c < kSsimRow && gj >= 0 && gj < W;
    }
    const uint32_t dst0 = (uint32_t)__cvta_generic_to_shared(&s[0][lane]);
    const float* src0 = img + ((int64_t)(v * (int64_t)H + (i0 - kSsimR)) * W + (j0 - kSsimR)) * 3 + lane;
    const int64_t row_stride = (int64_t)W * 3;
#pragma unroll
    for (int k = 0; k < (kSsimHalo + 7) / 8; ++k) {
        const int r = warp + 8 * k;
        if (r < kSsimHalo) {
            const int gi = i0 - kSsimR + r;
            const bool row_in = gi >= 0 && gi < H;
            const float* row = src0 + r * row_stride;
            const uint32_t drow = dst0 + (uint32_t)(r * ROW * 4);
#pragma unroll
            for (int it = 0; it < 3; ++it) {
                if (lane + 32 * it < kSsimRow) {
                    const bool in = row_in && col_in[it];
                    const float* src = in ? row + 32 * it : img;     // not read when the source size is 0
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(drow + 128 * it), "l"(src), "r"(in ? 4 : 0) : "memory");
                }
            }
        }
    }
}
__device__ __forceinline__ void halo_wait() {
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
    __syncthreads();
}

// ---- TMA halo loads (cp.async.bulk.tensor over a [C][H][W * 3] tensor map, box 1 x 26 x 80): one thread issues the copy of a
// whole halo tile, rows and columns outside the image are filled with zeros by the copy engine (= the zero padding of
// reading A21), completion is signalled on an mbarrier.
__device__ __forceinline__ void tma_init(uint64_t* mbar) {
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(mbar)), "r"(1) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
}
__device__ __forceinline__ void tma_expect(uint64_t* mbar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(mbar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_halo(const CUtensorMap* map, uint64_t* mbar, void* dst, int v, int i0, int j0) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"((j0 - kSsimR) * 3 - kSsimTmaOff), "r"(i0 - kSsimR),
                   "r"(v), "r"((uint32_t)__cvta_generic_to_shared(mbar))
                 : "memory");
}
__device__ __forceinline__ void tma_wait(uint64_t* mbar) {
    const uint32_t addr = (uint32_t)__cvta_generic_to_shared(mbar);
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.b32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(addr), "r"(0) : "memory");
    } while (!done);
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

// Both passes of the separable window keep a run of outputs in registers and stream over the inputs (4 outputs from 14
// inputs), so an input is read from shared memory once per run instead of once per tap; the three channels are processed
// together.  Horizontal tasks: (row, column group of 4, channel); vertical tasks: (row group of 4, column, channel) with
// the channel fastest, so that consecutive threads write consecutive addresses of the interleaved [.., 3] layout.
constexpr int kSsimRun = 4;
constexpr int kSsimIn = kSsimRun + kSsimWin - 1;        // 14 inputs feed 4 outputs
constexpr int kHzRow = kSsimTile + 1;

template <int Q>
struct HzBuf {
    // per-channel stride = 11 (mod 32) words: the vertical pass reads (channel, column) across a warp -> banks column + 11 channel
    static constexpr int kPad = (11 - (Q * kSsimHalo * kHzRow) % 32 + 32) % 32;
    float v[3][Q * kSsimHalo * kHzRow + kPad];
    __device__ __forceinline__ float& at(int ch, int q, int r, int c) { return v[ch][(q * kSsimHalo + r) * kHzRow + c]; }
};

template <bool TMA>
__global__ void __launch_bounds__(256) ssim_stats_kernel(const SsimArgs a, const __grid_constant__ CUtensorMap mx, const __grid_constant__ CUtensorMap my) {
    pdl_enter();
    constexpr int ROW = TMA ? kSsimRowTma : kSsimRowPad;
    constexpr int OFF = TMA ? kSsimTmaOff : 0;            // column of the halo's first float inside a staged row
    __shared__ __align__(128) float sx[kSsimHalo][ROW];
    __shared__ __align__(128) float sy[kSsimHalo][ROW];
    __shared__ HzBuf<5> hz;
    __shared__ float s_red[8];
    __shared__ uint64_t s_mbar;
    const int v = blockIdx.z, i0 = blockIdx.y * kSsimTile, j0 = blockIdx.x * kSsimTile;
    if constexpr (TMA) {
        tma_init(&s_mbar);
        if (threadIdx.x == 0) {
            tma_expect(&s_mbar, 2 * kSsimTmaBytes);
            tma_load_halo(&mx, &s_mbar, sx, v, i0, j0);
            tma_load_halo(&my, &s_mbar, sy, v, i0, j0);
        }
        tma_wait(&s_mbar);
    } else {
        load_halo_async<ROW>(a.x, v, i0, j0, a.H, a.W, sx);
        load_halo_async<ROW>(a.y, v, i0, j0, a.H, a.W, sy);
        halo_wait();
    }
    // horizontal pass
    for (int task = threadIdx.x; task < kSsimHalo * 3 * (kSsimTile / kSsimRun); task += 256) {
        const int r = task / 12, rem = task - r * 12, cg = rem / 3, ch = rem - cg * 3;
        // (x, y) and (x^2, y^2) travel as two-wide pairs: three instructions per tap and output instead of five
        f32x2 accA[kSsimRun], accB[kSsimRun];
        float accC[kSsimRun];
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) { accA[o] = pk2(0.f, 0.f); accB[o] = accA[o]; accC[o] = 0.0f; }
#pragma unroll
        for (int p = 0; p < kSsimIn; ++p) {
            const float xv = sx[r][(kSsimRun * cg + p) * 3 + ch + OFF], yv = sy[r][(kSsimRun * cg + p) * 3 + ch + OFF];
            const f32x2 X = pk2(xv, yv);
            const f32x2 P = mul2(X, X);
            const float xy = xv * yv;
#pragma unroll
            for (int o = 0; o < kSsimRun; ++o) {
                const int t = p - o;
                if (t >= 0 && t < kSsimWin) {
                    const float w = a.win[t];
                    const f32x2 W2 = pk2(w, w);
                    accA[o] = fma2(W2, X, accA[o]); accB[o] = fma2(W2, P, accB[o]); accC[o] = fmaf(w, xy, accC[o]);
                }
            }
        }
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) {
            float m1, m2, e11, e22;
            unpk2(accA[o], m1, m2); unpk2(accB[o], e11, e22);
            const int c = kSsimRun * cg + o;
            hz.at(ch, 0, r, c) = m1; hz.at(ch, 1, r, c) = m2; hz.at(ch, 2, r, c) = e11; hz.at(ch, 3, r, c) = e22; hz.at(ch, 4, r, c) = accC[o];
        }
    }
    __syncthreads();
    // vertical pass, SSIM and its derivatives
    const float wgt = -a.lambda * a.inv_n;
    float ssim_sum = 0.0f, l1_sum = 0.0f;
    if (threadIdx.x < 3 * kSsimTile * (kSsimTile / kSsimRun)) {
        const int ch = threadIdx.x % 3, col = (threadIdx.x / 3) % kSsimTile, g = threadIdx.x / (3 * kSsimTile);
        f32x2 accA[kSsimRun], accB[kSsimRun];
        float accC[kSsimRun];
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) { accA[o] = pk2(0.f, 0.f); accB[o] = accA[o]; accC[o] = 0.0f; }
#pragma unroll
        for (int p = 0; p < kSsimIn; ++p) {
            float in[5];
#pragma unroll
            for (int q = 0; q < 5; ++q) in[q] = hz.at(ch, q, kSsimRun * g + p, col);
            const f32x2 A2 = pk2(in[0], in[1]), B2 = pk2(in[2], in[3]);
#pragma unroll
            for (int o = 0; o < kSsimRun; ++o) {
                const int t = p - o;
                if (t >= 0 && t < kSsimWin) {
                    const float w = a.win[t];
                    const f32x2 W2 = pk2(w, w);
                    accA[o] = fma2(W2, A2, accA[o]); accB[o] = fma2(W2, B2, accB[o]); accC[o] = fmaf(w, in[4], accC[o]);
                }
            }
        }
        float acc[kSsimRun][5];
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) {
            unpk2(accA[o], acc[o][0], acc[o][1]); unpk2(accB[o], acc[o][2], acc[o][3]);
            acc[o][4] = accC[o];
        }
        const int gj = j0 + col;
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) {
            const int ty = kSsimRun * g + o, gi = i0 + ty;
            if (gi < a.H && gj < a.W) {
                const float mu1 = acc[o][0], mu2 = acc[o][1];
                const float s11 = acc[o][2] - mu1 * mu1, s22 = acc[o][3] - mu2 * mu2, s12 = acc[o][4] - mu1 * mu2;
                const float A1 = fmaf(2.0f * mu1, mu2, kSsimC1), A2 = fmaf(2.0f, s12, kSsimC2);
                const float B1 = fmaf(mu1, mu1, fmaf(mu2, mu2, kSsimC1)), B2 = s11 + s22 + kSsimC2;
                const float inv = 1.0f / (B1 * B2);
                const float S = A1 * A2 * inv;
                const float d11 = -S / B2;                                   // dS/ds11
                const float d12 = 2.0f * A1 * inv;                           // dS/ds12
                const float dmu = 2.0f * mu2 * A2 * inv - 2.0f * mu1 * S / B1 - 2.0f * mu1 * d11 - mu2 * d12;   // total dS/dmu1
                const int64_t o3 = 3 * (((int64_t)v * a.H + gi) * a.W + gj) + ch;
                a.maps[o3] = wgt * dmu;
                a.maps[a.n + o3] = wgt * d11;
                a.maps[2 * a.n + o3] = wgt * d12;
                ssim_sum += S;
                l1_sum += fabsf(sx[ty + kSsimR][(col + kSsimR) * 3 + ch + OFF] - sy[ty + kSsimR][(col + kSsimR) * 3 + ch + OFF]);
            }
        }
    }
    const float part = (1.0f - a.lambda) * l1_sum * a.inv_n - a.lambda * ssim_sum * a.inv_n;
    float tot = block_sum(part, s_red);
    if (threadIdx.x == 0) {
        if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) tot += a.lambda;     // the constant of lambda (1 - mean SSIM)
        atomicAdd(a.loss, tot);
    }
}

template <bool TMA>
__global__ void __launch_bounds__(256) ssim_grad_kernel(const SsimArgs a, const __grid_constant__ CUtensorMap m0, const __grid_constant__ CUtensorMap m1,
                                                        const __grid_constant__ CUtensorMap m2) {
    pdl_enter();
    constexpr int ROW = TMA ? kSsimRowTma : kSsimRowPad;
    constexpr int OFF = TMA ? kSsimTmaOff : 0;
    __shared__ __align__(128) float sm[3][kSsimHalo][ROW];
    __shared__ HzBuf<3> hz;
    __shared__ uint64_t s_mbar;
    const int v = blockIdx.z, i0 = blockIdx.y * kSsimTile, j0 = blockIdx.x * kSsimTile;
    if constexpr (TMA) {
        tma_init(&s_mbar);
        if (threadIdx.x == 0) {
            tma_expect(&s_mbar, 3 * kSsimTmaBytes);
            tma_load_halo(&m0, &s_mbar, sm[0], v, i0, j0);
            tma_load_halo(&m1, &s_mbar, sm[1], v, i0, j0);
            tma_load_halo(&m2, &s_mbar, sm[2], v, i0, j0);
        }
    } else {
#pragma unroll
        for (int q = 0; q < 3; ++q) load_halo_async<ROW>(a.maps + q * a.n, v, i0, j0, a.H, a.W, sm[q]);
    }
    // x and y at this thread's four output values travel while the window passes run
    const bool vtask = threadIdx.x < 3 * kSsimTile * (kSsimTile / kSsimRun);
    const int vch = threadIdx.x % 3, vcol = (threadIdx.x / 3) % kSsimTile, vg = threadIdx.x / (3 * kSsimTile);
    float xo[kSsimRun], yo[kSsimRun];
#pragma unroll
    for (int o = 0; o < kSsimRun; ++o) {
        const int gi = i0 + kSsimRun * vg + o, gj = j0 + vcol;
        xo[o] = 0.0f; yo[o] = 0.0f;
        if (vtask && gi < a.H && gj < a.W) {
            const int64_t o3 = 3 * (((int64_t)v * a.H + gi) * a.W + gj) + vch;
            xo[o] = __ldg(a.x + o3); yo[o] = __ldg(a.y + o3);
        }
    }
    if constexpr (TMA) tma_wait(&s_mbar);
    else halo_wait();
    for (int task = threadIdx.x; task < kSsimHalo * 3 * (kSsimTile / kSsimRun); task += 256) {
        const int r = task / 12, rem = task - r * 12, cg = rem / 3, ch = rem - cg * 3;
        f32x2 accA[kSsimRun];
        float accC[kSsimRun];
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) { accA[o] = pk2(0.f, 0.f); accC[o] = 0.0f; }
#pragma unroll
        for (int p = 0; p < kSsimIn; ++p) {
            float in[3];
#pragma unroll
            for (int q = 0; q < 3; ++q) in[q] = sm[q][r][(kSsimRun * cg + p) * 3 + ch + OFF];
            const f32x2 A2 = pk2(in[0], in[1]);
#pragma unroll
            for (int o = 0; o < kSsimRun; ++o) {
                const int t = p - o;
                if (t >= 0 && t < kSsimWin) {
                    const float w = a.win[t];
                    accA[o] = fma2(pk2(w, w), A2, accA[o]); accC[o] = fmaf(w, in[2], accC[o]);
                }
            }
        }
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) {
            float g0, g1;
            unpk2(accA[o], g0, g1);
            const int c = kSsimRun * cg + o;
            hz.at(ch, 0, r, c) = g0; hz.at(ch, 1, r, c) = g1; hz.at(ch, 2, r, c) = accC[o];
        }
    }
    __syncthreads();
    if (vtask) {
        const int ch = vch, col = vcol, g = vg;
        f32x2 accA[kSsimRun];
        float accC[kSsimRun];
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) { accA[o] = pk2(0.f, 0.f); accC[o] = 0.0f; }
#pragma unroll
        for (int p = 0; p < kSsimIn; ++p) {
            float in[3];
#pragma unroll
            for (int q = 0; q < 3; ++q) in[q] = hz.at(ch, q, kSsimRun * g + p, col);
            const f32x2 A2 = pk2(in[0], in[1]);
#pragma unroll
            for (int o = 0; o < kSsimRun; ++o) {
                const int t = p - o;
                if (t >= 0 && t < kSsimWin) {
                    const float w = a.win[t];
                    accA[o] = fma2(pk2(w, w), A2, accA[o]); accC[o] = fmaf(w, in[2], accC[o]);
                }
            }
        }
        float acc[kSsimRun][3];
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) { unpk2(accA[o], acc[o][0], acc[o][1]); acc[o][2] = accC[o]; }
        const float l1w = (1.0f - a.lambda) * a.inv_n;
        const int gj = j0 + col;
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) {
            const int gi = i0 + kSsimRun * g + o;
            if (gi < a.H && gj < a.W) {
                const int64_t o3 = 3 * (((int64_t)v * a.H + gi) * a.W + gj) + ch;
                const float xv = xo[o], yv = yo[o];
                const float d = xv - yv;
                const float l1 = d > 0.f ? l1w : (d < 0.f ? -l1w : 0.f);
                a.dL[o3] = fmaf(2.0f * xv, acc[o][1], fmaf(yv, acc[o][2], acc[o][0])) + l1;
            }
        }
    }
}

// cuTensorMapEncodeTiled through the runtime's driver entry point query (no link-time dependency on libcuda: the library
// must load on a machine without a driver); nullptr when unavailable -> the cp.async path is used
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn tensor_map_encoder() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;          // idempotent cache of an immutable fact, like DeviceCache
    if (!tried) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
        tried = true;
    }
    return fn;
}
// [C][H][W * 3] fp32 image as a 3-D tensor, box = one view x 26 rows x 80 floats, zero fill outside
static bool make_halo_map(EncodeTiledFn enc, const float* img, int C, int H, int W, CUtensorMap* out) {
    const cuuint64_t dims[3] = {(cuuint64_t)W * 3, (cuuint64_t)H, (cuuint64_t)C};
    const cuuint64_t strides[2] = {(cuuint64_t)W * 3 * sizeof(float), (cuuint64_t)H * W * 3 * sizeof(float)};
    const cuuint32_t box[3] = {(cuuint32_t)kSsimRowTma, (cuuint32_t)kSsimHalo, 1u};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    return enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(img), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
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
    // TMA halo loads need 16-byte aligned images and row strides (W % 4 == 0); everything else takes the cp.async path
    CUtensorMap mx, my, m0, m1, m2;
    bool tma = false;
    if (width % 4 == 0 && aligned(image, 16) && aligned(target, 16) && aligned(workspace, 16) && n % 4 == 0) {
        if (EncodeTiledFn enc = tensor_map_encoder())
            tma = make_halo_map(enc, image, C, height, width, &mx) && make_halo_map(enc, target, C, height, width, &my) &&
                  make_halo_map(enc, a.maps, C, height, width, &m0) && make_halo_map(enc, a.maps + n, C, height, width, &m1) &&
                  make_halo_map(enc, a.maps + 2 * n, C, height, width, &m2);
    }
    if (tma) launch_chained(ssim_stats_kernel<true>, dim3(grid), dim3(256), (size_t)(0), st, a, mx, my);
    else launch_chained(ssim_stats_kernel<false>, dim3(grid), dim3(256), (size_t)(0), st, a, mx, my);
    int rc = launch_status();
    if (rc) return rc;
    if (tma) launch_chained(ssim_grad_kernel<true>, dim3(grid), dim3(256), (size_t)(0), st, a, m0, m1, m2);
    else launch_chained(ssim_grad_kernel<false>, dim3(grid), dim3(256), (size_t)(0), st, a, m0, m1, m2);
    return launch_status();
}
