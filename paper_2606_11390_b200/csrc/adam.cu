// adam.cu -- fused Adam step over one parameter array of the Gaussians.
// m <- b1 m + (1 - b1) g;  v <- b2 v + (1 - b2) g^2;  p <- p - lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps)
// (readings A27, A28).  One streaming pass: 16 bytes read and 12 written per element, 16-byte accesses.  With the saved
// radii[C, N] the "visible-only" variant touches only the rows of Gaussians visible in >= 1 view of the batch: at street
// scale that is a fraction of a per cent of the 28 x 59 bytes per Gaussian.
#include "common.cuh"

namespace gs {

struct AdamArgs {
    int64_t N;
    int32_t row;            // floats per Gaussian in this array
    float* p; const float* g; float* m; float* v;
    float lr, b1, b2, eps, c1, c2;      // c1 = 1 / (1 - b1^t), c2 = 1 / (1 - b2^t)
    const int32_t* radii; int32_t C;
    float* running_max;     // optional: max over the updated parameter values
};

// max for floats of either sign through the integer atomics (NaNs are not recorded)
__device__ __forceinline__ void atomic_max_float(float* addr, float v) {
    if (v >= 0.0f) atomicMax(reinterpret_cast<int*>(addr), __float_as_int(v));
    else if (v < 0.0f) atomicMin(reinterpret_cast<unsigned int*>(addr), __float_as_uint(v));
}

__device__ __forceinline__ void warp_running_max(float* running_max, float vmax) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, d));
    if ((threadIdx.x & 31) == 0 && vmax > -3.0e38f) atomic_max_float(running_max, vmax);
}

__device__ __forceinline__ void adam1(float& p, float g, float& m, float& v, const AdamArgs& a) {
    m = fmaf(a.b1, m, (1.0f - a.b1) * g);
    v = fmaf(a.b2, v, (1.0f - a.b2) * g * g);
    p -= a.lr * (m * a.c1) / (sqrtf(v * a.c2) + a.eps);
}

// dense: one thread per 16-byte unit
__global__ void __launch_bounds__(256) adam_dense_kernel(const AdamArgs a, int64_t n4, int64_t n) {
    pdl_enter();
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    float vmax = -3.0e38f;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n4; k += stride) {
        float4 p = reinterpret_cast<float4*>(a.p)[k], m = reinterpret_cast<float4*>(a.m)[k], v = reinterpret_cast<float4*>(a.v)[k];
        const float4 g = __ldg(reinterpret_cast<const float4*>(a.g) + k);
        adam1(p.x, g.x, m.x, v.x, a); adam1(p.y, g.y, m.y, v.y, a); adam1(p.z, g.z, m.z, v.z, a); adam1(p.w, g.w, m.w, v.w, a);
        reinterpret_cast<float4*>(a.p)[k] = p; reinterpret_cast<float4*>(a.m)[k] = m; reinterpret_cast<float4*>(a.v)[k] = v;
        vmax = fmaxf(vmax, fmaxf(fmaxf(p.x, p.y), fmaxf(p.z, p.w)));
    }
    if (blockIdx.x == 0 && threadIdx.x < (int)(n - 4 * n4)) {
        const int64_t k = 4 * n4 + threadIdx.x;
        float p = a.p[k], m = a.m[k], v = a.v[k];
        adam1(p, a.g[k], m, v, a);
        a.p[k] = p; a.m[k] = m; a.v[k] = v;
        vmax = fmaxf(vmax, p);
    }
    if (a.running_max) warp_running_max(a.running_max, vmax);
}

// scalar fall-back for unaligned arrays, and the visible-only variant: a warp scans 32 Gaussians' radii over the C views
// and then walks the visible rows, lanes across the row's floats
__global__ void __launch_bounds__(256) adam_rows_kernel(const AdamArgs a) {
    pdl_enter();
    const int lane = threadIdx.x & 31;
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    float vmax = -3.0e38f;
    for (int64_t base = warp * 32; base < a.N; base += nwarps * 32) {
        const int64_t i = base + lane;
        bool vis = false;
        if (i < a.N) {
            vis = a.radii == nullptr;
            for (int c = 0; c < a.C && !vis; ++c) vis = __ldg(a.radii + (int64_t)c * a.N + i) > 0;
        }
        unsigned int mask = __ballot_sync(0xffffffffu, vis);
        while (mask) {
            const int s = __ffs(mask) - 1;
            mask &= mask - 1;
            const int64_t r0 = (base + s) * a.row;
            for (int k = lane; k < a.row; k += 32) {
                float p = a.p[r0 + k], m = a.m[r0 + k], v = a.v[r0 + k];
                adam1(p, __ldg(a.g + r0 + k), m, v, a);
                a.p[r0 + k] = p; a.m[r0 + k] = m; a.v[r0 + k] = v;
                vmax = fmaxf(vmax, p);
            }
        }
    }
    if (a.running_max) warp_running_max(a.running_max, vmax);
}

// Visible-only step over up to 8 arrays at once: the radii are scanned ONCE (16-byte loads, 4 Gaussians per lane and view),
// then the warp walks the visible Gaussians and, for each, the rows of all arrays with the lanes across the floats.
constexpr int kAdamMaxArrays = 8;
struct AdamMultiArgs {
    int64_t N;
    int32_t n_arrays, C, vec;
    int32_t row[kAdamMaxArrays];
    int32_t start[kAdamMaxArrays];      // first element of array q in the concatenated row
    int32_t total_row;
    float* p[kAdamMaxArrays]; const float* g[kAdamMaxArrays]; float* m[kAdamMaxArrays]; float* v[kAdamMaxArrays];
    float lr, b1, b2, eps, c1, c2;
    const int32_t* radii;
    const uint32_t* vmask;      // alternative to radii: the visibility mask [C][wn] of gs_project_fwd
    int64_t wn;
    float* running_max;         // optional: *running_max = max(*running_max, every updated value of array max_array)
    int32_t max_array;
};

// the rows of one visible Gaussian in all arrays: the lanes run over the concatenation of the rows (59 floats for the five
// parameter arrays at SH degree 3), every load of a Gaussian is issued before the first use
__device__ __forceinline__ void adam_gaussian(const AdamMultiArgs& a, const AdamArgs& h, int64_t i, int lane, float& vmax) {
    for (int e = lane; e < a.total_row; e += 32) {
        int q = 0;
#pragma unroll
        for (int j = 1; j < kAdamMaxArrays; ++j) q += (j < a.n_arrays && e >= a.start[j]) ? 1 : 0;
        const int64_t o = i * a.row[q] + (e - a.start[q]);
        float p = a.p[q][o], m = a.m[q][o], v = a.v[q][o];
        adam1(p, __ldg(a.g[q] + o), m, v, h);
        a.p[q][o] = p; a.m[q][o] = m; a.v[q][o] = v;
        if (q == a.max_array) vmax = fmaxf(vmax, p);
    }
}

__global__ void __launch_bounds__(256) adam_visible_multi_kernel(const AdamMultiArgs a) {
    pdl_enter();
    const int lane = threadIdx.x & 31;
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    AdamArgs h;
    h.lr = a.lr; h.b1 = a.b1; h.b2 = a.b2; h.eps = a.eps; h.c1 = a.c1; h.c2 = a.c2;
    float vmax = -3.0e38f;
    if (a.vmask) {
        // one mask word (32 Gaussians) per lane and view; the warp then walks the set bits of the non-zero words
        for (int64_t base = warp * 1024; base < a.N; base += nwarps * 1024) {
            const int64_t word = (base >> 5) + lane;
            unsigned int vis = 0;
            if (word < a.wn)
                for (int c = 0; c < a.C; ++c) vis |= __ldg(a.vmask + (int64_t)c * a.wn + word);
            unsigned int nz = __ballot_sync(0xffffffffu, vis != 0u);
            while (nz) {
                const int s = __ffs(nz) - 1;
                nz &= nz - 1;
                unsigned int bits = __shfl_sync(0xffffffffu, vis, s);
                while (bits) {
                    const int b = __ffs(bits) - 1;
                    bits &= bits - 1;
                    adam_gaussian(a, h, base + 32 * s + b, lane, vmax);
                }
            }
        }
    } else {
        for (int64_t base = warp * 128; base < a.N; base += nwarps * 128) {
            const int64_t i0 = base + 4 * lane;
            unsigned int vis = 0;                       // bit k: Gaussian i0 + k is visible in some view
            for (int c = 0; c < a.C; ++c) {
                const int32_t* r = a.radii + (int64_t)c * a.N + i0;
                if (a.vec && i0 + 4 <= a.N) {
                    const int4 q = __ldg(reinterpret_cast<const int4*>(r));
                    vis |= (q.x > 0 ? 1u : 0u) | (q.y > 0 ? 2u : 0u) | (q.z > 0 ? 4u : 0u) | (q.w > 0 ? 8u : 0u);
                } else {
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        if (i0 + k < a.N && __ldg(r + k) > 0) vis |= 1u << k;
                }
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                unsigned int mask = __ballot_sync(0xffffffffu, (vis >> k) & 1u);
                while (mask) {
                    const int s = __ffs(mask) - 1;
                    mask &= mask - 1;
                    adam_gaussian(a, h, base + 4 * s + k, lane, vmax);
                }
            }
        }
    }
    if (a.running_max) warp_running_max(a.running_max, vmax);
}

}  // namespace gs

using namespace gs;

extern "C" int gs_adam_step_visible(int64_t N, int32_t n_arrays, const int32_t* row_floats, float* const* params, const float* const* grads,
                                    float* const* ms, float* const* vs, float lr, float beta1, float beta2, float eps, int32_t step,
                                    const int32_t* radii, const uint32_t* vis_mask, int32_t C, float* running_max, int32_t max_array,
                                    void* stream) {
    if (N < 0 || n_arrays < 1 || n_arrays > kAdamMaxArrays || step < 1 || !row_floats || !params || !grads || !ms || !vs) return GS_ERR_INVALID_ARGUMENT;
    if (!(beta1 >= 0.0f && beta1 < 1.0f) || !(beta2 >= 0.0f && beta2 < 1.0f) || !finite_f(lr) || !(eps >= 0.0f)) return GS_ERR_INVALID_ARGUMENT;
    if ((!radii && !vis_mask) || C < 1 || C > GS_MAX_VIEWS) return GS_ERR_INVALID_ARGUMENT;
    if (running_max && (max_array < 0 || max_array >= n_arrays)) return GS_ERR_INVALID_ARGUMENT;
    if (N == 0) return GS_OK;
    AdamMultiArgs a;
    a.N = N; a.n_arrays = n_arrays; a.C = C; a.radii = radii;
    a.vmask = vis_mask; a.wn = GS_VIS_WORDS(N);
    a.running_max = running_max; a.max_array = running_max ? max_array : -1;
    a.vec = (radii && aligned(radii, 16) && (N % 4 == 0 || C == 1)) ? 1 : 0;
    a.total_row = 0;
    for (int q = 0; q < kAdamMaxArrays; ++q) { a.row[q] = 1; a.start[q] = 0; a.p[q] = nullptr; a.g[q] = nullptr; a.m[q] = nullptr; a.v[q] = nullptr; }
    for (int q = 0; q < n_arrays; ++q) {
        if (row_floats[q] < 1 || row_floats[q] > 4096 || !params[q] || !grads[q] || !ms[q] || !vs[q]) return GS_ERR_INVALID_ARGUMENT;
        a.row[q] = row_floats[q]; a.p[q] = params[q]; a.g[q] = grads[q]; a.m[q] = ms[q]; a.v[q] = vs[q];
        a.start[q] = a.total_row;
        a.total_row += row_floats[q];
    }
    a.lr = lr; a.b1 = beta1; a.b2 = beta2; a.eps = eps;
    a.c1 = (float)(1.0 / (1.0 - pow((double)beta1, (double)step)));
    a.c2 = (float)(1.0 / (1.0 - pow((double)beta2, (double)step)));
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    int64_t blocks = (N + 1023) / 1024;
    if (blocks > (int64_t)sms * 8) blocks = (int64_t)sms * 8;
    launch_chained(adam_visible_multi_kernel, dim3((unsigned)blocks), dim3(256), (size_t)(0), (cudaStream_t)stream, a);
    return launch_status();
}


extern "C" int gs_adam_step(int64_t N, int32_t row_floats, float* param, const float* grad, float* m, float* v, float lr, float beta1,
                            float beta2, float eps, int32_t step, const int32_t* radii, int32_t C, float* running_max, void* stream) {
    if (N < 0 || row_floats < 1 || row_floats > 4096 || step < 1) return GS_ERR_INVALID_ARGUMENT;
    if (!(beta1 >= 0.0f && beta1 < 1.0f) || !(beta2 >= 0.0f && beta2 < 1.0f) || !finite_f(lr) || !(eps >= 0.0f)) return GS_ERR_INVALID_ARGUMENT;
    if (radii && (C < 1 || C > GS_MAX_VIEWS)) return GS_ERR_INVALID_ARGUMENT;
    if (N == 0) return GS_OK;
    if (!param || !grad || !m || !v) return GS_ERR_INVALID_ARGUMENT;
    AdamArgs a;
    a.N = N; a.row = row_floats; a.p = param; a.g = grad; a.m = m; a.v = v;
    a.lr = lr; a.b1 = beta1; a.b2 = beta2; a.eps = eps;
    a.c1 = (float)(1.0 / (1.0 - pow((double)beta1, (double)step)));
    a.c2 = (float)(1.0 / (1.0 - pow((double)beta2, (double)step)));
    a.radii = radii; a.C = radii ? C : 0; a.running_max = running_max;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n = N * row_floats;
    if (!radii && aligned(param, 16) && aligned(grad, 16) && aligned(m, 16) && aligned(v, 16)) {
        const int64_t n4 = n >> 2;
        int64_t blocks = (n4 + 255) / 256;
        if (blocks > (int64_t)sms * 32) blocks = (int64_t)sms * 32;
        launch_chained(adam_dense_kernel, dim3((unsigned)(blocks < 1 ? 1 : blocks)), dim3(256), (size_t)(0), st, a, n4, n);
    } else {
        int64_t blocks = (N + 255) / 256;
        if (blocks > (int64_t)sms * 16) blocks = (int64_t)sms * 16;
        launch_chained(adam_rows_kernel, dim3((unsigned)blocks), dim3(256), (size_t)(0), st, a);
    }
    return launch_status();
}
