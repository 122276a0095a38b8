// morton.cu -- 3-D Morton ordering of the Gaussian arrays ("sorted along a Morton
// curve").  Steps: gs_bounds (bounding box of the means) -> gs_morton_codes (21 bits per axis, interleaved to 63 bits)
// -> gs_sort_pairs (binning.cu's stable radix sort on the codes, values = indices) -> gs_gather_rows (apply the
// permutation to every parameter array).  Readings A24-A26 in DESIGN.md.
#include "common.cuh"

namespace gs {

// order-preserving map float -> uint32 (and back), so that atomicMin / atomicMax on the integers order the floats
__device__ __forceinline__ unsigned int f2ord(float f) {
    const unsigned int u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(unsigned int o) {
    return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}

__global__ void bounds_init_kernel(unsigned int* b) {
    pdl_enter();
    if (threadIdx.x < 3) b[threadIdx.x] = 0xffffffffu;          // running minimum
    else if (threadIdx.x < 6) b[threadIdx.x] = 0u;               // running maximum
}
__global__ void __launch_bounds__(256) bounds_kernel(int64_t N, const float* __restrict__ means, unsigned int* b) {
    pdl_enter();
    unsigned int lo[3] = {0xffffffffu, 0xffffffffu, 0xffffffffu}, hi[3] = {0u, 0u, 0u};
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const unsigned int o = f2ord(__ldg(means + 3 * i + k));
            lo[k] = min(lo[k], o); hi[k] = max(hi[k], o);
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            lo[k] = min(lo[k], __shfl_xor_sync(0xffffffffu, lo[k], d));
            hi[k] = max(hi[k], __shfl_xor_sync(0xffffffffu, hi[k], d));
        }
        if ((threadIdx.x & 31) == 0) { atomicMin(b + k, lo[k]); atomicMax(b + 3 + k, hi[k]); }
    }
}
__global__ void bounds_decode_kernel(unsigned int* b) {
    pdl_enter();
    if (threadIdx.x < 6) {
        const float f = ord2f(b[threadIdx.x]);
        reinterpret_cast<float*>(b)[threadIdx.x] = f;
    }
}

// spread the low 21 bits of x so that bit k lands at bit 3k
__device__ __forceinline__ unsigned long long spread3(unsigned long long x) {
    x &= 0x1fffffull;
    x = (x | (x << 32)) & 0x1f00000000ffffull;
    x = (x | (x << 16)) & 0x1f0000ff0000ffull;
    x = (x | (x << 8)) & 0x100f00f00f00f00full;
    x = (x | (x << 4)) & 0x10c30c30c30c30c3ull;
    x = (x | (x << 2)) & 0x1249249249249249ull;
    return x;
}

__global__ void __launch_bounds__(256) morton_codes_kernel(int64_t N, const float* __restrict__ means, const float* __restrict__ lo_hi,
                                                           unsigned long long* __restrict__ codes, int32_t* __restrict__ index) {
    pdl_enter();
    float lo[3], sc[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        lo[k] = __ldg(lo_hi + k);
        const float ext = __fsub_rn(__ldg(lo_hi + 3 + k), lo[k]);
        sc[k] = ext > 0.0f ? __fdiv_rn(2097152.0f, ext) : 1.0f;
    }
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
        unsigned long long q[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            // one rounding per operation (reading A24): no FMA contraction
            float t = floorf(__fmul_rn(__fsub_rn(__ldg(means + 3 * i + k), lo[k]), sc[k]));
            if (!(fabsf(t) < CUDART_INF_F)) t = 0.0f;            // NaN or infinite
            t = fminf(fmaxf(t, 0.0f), 2097151.0f);
            q[k] = (unsigned long long)t;
        }
        codes[i] = (spread3(q[0]) << 2) | (spread3(q[1]) << 1) | spread3(q[2]);
        index[i] = (int32_t)i;
    }
}

// dst[i, :] = src[perm[i], :]; one thread per 16-byte unit when the rows allow it
template <typename T>
__global__ void __launch_bounds__(256) gather_rows_kernel(int64_t N, int units, const T* __restrict__ src, const int32_t* __restrict__ perm,
                                                          T* __restrict__ dst) {
    pdl_enter();
    const int64_t total = N * units;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = k / units;
        const int u = (int)(k - i * units);
        dst[k] = __ldg(src + (int64_t)__ldg(perm + i) * units + u);
    }
}

static unsigned grid_for(int64_t items) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int64_t blocks = (items + 255) / 256;
    const int64_t cap = (int64_t)sms * 16;
    return (unsigned)(blocks < 1 ? 1 : (blocks < cap ? blocks : cap));
}

}  // namespace gs

using namespace gs;

extern "C" int gs_bounds(int64_t N, const float* means, float* lo_hi, void* stream) {
    if (N < 1 || !means || !lo_hi || !aligned(lo_hi, 4)) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned int* b = reinterpret_cast<unsigned int*>(lo_hi);
    launch_chained(bounds_init_kernel, dim3(1), dim3(32), (size_t)(0), st, b);
    launch_chained(bounds_kernel, dim3(grid_for(N)), dim3(256), (size_t)(0), st, N, means, b);
    launch_chained(bounds_decode_kernel, dim3(1), dim3(32), (size_t)(0), st, b);
    return launch_status();
}

extern "C" int gs_morton_codes(int64_t N, const float* means, const float* lo_hi, uint64_t* codes, int32_t* index, void* stream) {
    if (N < 0 || N >= (1LL << 31)) return GS_ERR_INVALID_ARGUMENT;
    if (N == 0) return GS_OK;
    if (!means || !lo_hi || !codes || !index || !aligned(codes, 8)) return GS_ERR_INVALID_ARGUMENT;
    launch_chained(morton_codes_kernel, dim3(grid_for(N)), dim3(256), (size_t)(0), (cudaStream_t)stream, N, means, lo_hi, reinterpret_cast<unsigned long long*>(codes), index);
    return launch_status();
}

extern "C" int gs_gather_rows(int64_t N, int32_t row_floats, const float* src, const int32_t* perm, float* dst, void* stream) {
    if (N < 0 || row_floats < 1 || row_floats > 4096) return GS_ERR_INVALID_ARGUMENT;
    if (N == 0) return GS_OK;
    if (!src || !perm || !dst || src == dst) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t st = (cudaStream_t)stream;
    if (row_floats % 4 == 0 && aligned(src, 16) && aligned(dst, 16))
        launch_chained(gather_rows_kernel<float4>, dim3(grid_for(N * (row_floats / 4))), dim3(256), (size_t)(0), st, N, row_floats / 4, reinterpret_cast<const float4*>(src), perm,
                                                                                  reinterpret_cast<float4*>(dst));
    else
        launch_chained(gather_rows_kernel<float>, dim3(grid_for(N * row_floats)), dim3(256), (size_t)(0), st, N, row_floats, src, perm, dst);
    return launch_status();
}
