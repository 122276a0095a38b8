// project.cu -- per-Gaussian stages P1 (gs_project_fwd) and P5 (gs_project_bwd) for sm_100a.
//
// The C views of the batch are looped inside one thread per Gaussian so that the parameters (236 B
// at SH degree 3) are read once for all cameras ("outputs colors and projected
// geometric quantities for all cameras in the batch").  Both kernels are persistent; every WARP works
// on its own chunks of consecutive Gaussians, independently of the other warps (no block barrier), in two phases:
//   phase A (streaming, every thread, vector loads/stores): P1 reads the 12-byte means (4 Gaussians =
//     3 x 16 B per thread), applies the near/far test of every view and zero-fills the chunk's radii /
//     tiles_touched; P5 reads the saved radii and zero-fills the chunk's rows of the five dense
//     gradient arrays with fully coalesced 16-byte stores.  The surviving Gaussians are pushed
//     onto a shared-memory stack that is carried across chunks;
//   phase B (runs whenever a full block of survivors is waiting, one thread each, so its warps are
//     fully populated even when a few per cent of the Gaussians survive): P1 first drops the views
//     whose tile rectangle must be empty from the mean and the largest scale alone (B0), then reads
//     rotation and the SH coefficients only for Gaussians that can be visible (B1); P5 evaluates the
//     chain rule for the visible Gaussians.
// So the HBM traffic is 12 N + 224 V_any + 48 sum_c V_c + 8 N C for P1 and 4 N C + 36 sum_c V_c +
// 236 V_any + 236 N for P5 ("algorithmic bytes"), and in the city/block regime (a few
// per cent visible) nearly all of it moves in phase A at full memory-level parallelism.
#include "project_math.cuh"

namespace gs {

struct ProjFwdArgs {
    int64_t N;
    int32_t C;
    const float* means; const float* log_scales; const float* quats; const float* logits; const float* sh;
    float* means2d; float* depths; float* conics; float* opacities; float* rgbs;
    int32_t* radii; uint32_t* tiles;
    float dilation, extent;
    int32_t vec_in, vec_out;   // 16-byte vector access allowed on means / on radii+tiles rows
    uint32_t* vmask;           // optional visibility mask [C][wn] (bit i & 31 of word i >> 5); replaces the dense zero-fill of radii / tiles
    int64_t wn;                // mask words per view, GS_VIS_WORDS(N)
    const float* ls_bound;     // optional device scalar >= every log-scale: the streaming phase then culls laterally as well
};

constexpr int kProjThreads = 128;   // P1 block
constexpr int kBwdThreads = 128;    // P5 block (168 registers per thread)
constexpr int64_t kZeroFillMinN = 1 << 22;   // from here the dense zero-fill of P5 runs as its own streaming kernels (measured:
                                             // slower at 1 M Gaussians, 0.555 -> 0.44 ms at 10 M, 2.98 -> 2.34 ms at 60 M)
constexpr int kProjItems = 8;   // Gaussians per thread in P1's streaming phase

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

// A warp's shared-memory stack of pending Gaussians: index, view mask and (P1 only) the mean, so that
// the later phases do not read it from memory again.  CAP entries per warp.
template <int CAP, bool WITH_MEAN>
struct WarpStack {
    uint32_t idx[CAP];
    uint32_t msk[CAP];
    float xyz[WITH_MEAN ? 3 : 1][WITH_MEAN ? CAP : 1];
};

// Warp-wide push of the items with a non-zero mask; `cnt` (the stack height) is warp-uniform.  The
// order is irrelevant: every output is addressed by the index.
template <int ITEMS, int CAP, bool WITH_MEAN>
__device__ __forceinline__ void warp_push(const uint32_t (&idx)[ITEMS], const uint32_t (&msk)[ITEMS], const float* m /*[3*ITEMS] or null*/,
                                          WarpStack<CAP, WITH_MEAN>& st, int& cnt, int lane) {
    if constexpr (ITEMS == 1) {
        const unsigned int b = __ballot_sync(0xffffffffu, msk[0] != 0u);
        if (msk[0]) {
            const int p = cnt + __popc(b & ((1u << lane) - 1u));
            st.idx[p] = idx[0];
            st.msk[p] = msk[0];
            if (WITH_MEAN) { st.xyz[0][p] = m[0]; st.xyz[WITH_MEAN ? 1 : 0][p] = m[1]; st.xyz[WITH_MEAN ? 2 : 0][p] = m[2]; }
        }
        cnt += __popc(b);
    } else {
        // several items per lane: one warp scan of the per-lane counts instead of one ballot per item; a lane's survivors
        // take consecutive slots
        int n = 0;
#pragma unroll
        for (int k = 0; k < ITEMS; ++k) n += msk[k] != 0u;
        int incl = n;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        int p = cnt + incl - n;
#pragma unroll
        for (int k = 0; k < ITEMS; ++k)
            if (msk[k]) {
                st.idx[p] = idx[k];
                st.msk[p] = msk[k];
                if (WITH_MEAN) { st.xyz[0][p] = m[3 * k]; st.xyz[WITH_MEAN ? 1 : 0][p] = m[3 * k + 1]; st.xyz[WITH_MEAN ? 2 : 0][p] = m[3 * k + 2]; }
                ++p;
            }
        cnt += __shfl_sync(0xffffffffu, incl, 31);
    }
}

// phase B of P1 for one Gaussian inside the depth range of the views in zmask
template <int DEG>
__device__ __forceinline__ void project_fwd_one(const ProjFwdArgs& a, const CamBatch& cams, int64_t i, uint32_t zmask, float px, float py,
                                                float pz) {
    uint32_t vis = 0;
    {
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
            if (a.vmask) atomicOr(a.vmask + (int64_t)c * a.wn + (i >> 5), 1u << (unsigned)(i & 31));
        }
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

// Conservative screen-space pre-cull from the mean and an upper bound of the largest scale alone (no rotation needed):
// |Sigma'| <= (s_max |J|_F |W|_2)^2 =: L, so lambda_max <= 2 (L + dilation) + sqrt(0.1) and the integer radius
// is at most rb = extent sqrt(that) + 1.  A view whose tile rectangle must then be empty (mean more
// than rb outside the 16-pixel-padded image) is dropped; phase B would cull it at step 8
// anyway, so no result changes.  Non-finite intermediates fail every comparison and keep the view.
// smax2 = (upper bound of the scale)^2; tz = the camera-space depth already computed by the caller.
__device__ __forceinline__ bool lateral_keep(const ProjFwdArgs& a, const DevCam& cam, float smax2, float px, float py, float pz, float tz) {
    const float tx = cam.W[0] * px + cam.W[1] * py + cam.W[2] * pz + cam.tau[0];
    const float ty = cam.W[3] * px + cam.W[4] * py + cam.W[5] * pz + cam.tau[1];
    const float rz = 1.0f / tz;
    const float u = cam.fx * tx * rz + cam.cx, v = cam.fy * ty * rz + cam.cy;
    const float jf = (cam.fx * cam.fx * (1.0f + cam.lim_x * cam.lim_x) + cam.fy * cam.fy * (1.0f + cam.lim_y * cam.lim_y)) * cam.wnorm2 * rz * rz;
    const float L = smax2 * jf;
    const float rb = a.extent * sqrtf(2.0f * (L + fmaxf(a.dilation, 0.0f)) + 0.32f) * 1.001f + 3.0f;
    const float w16 = (float)(cam.gx * kTile), h16 = (float)(cam.gy * kTile);
    const bool out = (u + rb + 16.0f < 0.0f) || (u - rb > w16) || (v + rb + 16.0f < 0.0f) || (v - rb > h16);
    return !out;
}
__device__ __forceinline__ uint32_t lateral_precull(const ProjFwdArgs& a, const CamBatch& cams, float lmax, float px, float py, float pz,
                                                    uint32_t zmask) {
    const float smax = expf(lmax);
    uint32_t keep = 0;
    for (int c = 0; c < a.C; ++c) {
        if (!((zmask >> c) & 1u)) continue;
        const DevCam& cam = cams.cam[c];
        const float tz = cam.W[6] * px + cam.W[7] * py + cam.W[8] * pz + cam.tau[2];
        if (lateral_keep(a, cam, smax * smax, px, py, pz, tz)) keep |= 1u << c;
    }
    return keep;
}

// Camera constants of the linear lateral test in shared memory (20 floats per view): the lanes of a warp test different
// views, and a lane-varying index into the constant bank would be replayed once per distinct view.
constexpr int kLatFloats = 20;
__device__ __forceinline__ void load_lateral_constants(const CamBatch& cams, int C, float smax_all, float (*s_lat)[kLatFloats]) {
    for (int k = threadIdx.x; k < C * kLatFloats; k += blockDim.x) {
        const int c = k / kLatFloats, j = k - c * kLatFloats;
        const DevCam& cam = cams.cam[c];
        float v = 0.0f;
        if (j < 9) v = cam.W[j];
        else if (j < 12) v = cam.tau[j - 9];
        else if (j == 12) v = cam.fx;
        else if (j == 13) v = cam.fy;
        else if (j == 14) v = cam.lat_cx;
        else if (j == 15) v = cam.lat_cy;
        else if (j == 16) v = cam.lat_k1x;
        else if (j == 17) v = cam.lat_k1y;
        else if (j == 18) v = fmaf(cam.lat_k2, smax_all, cam.lat_abs);
        s_lat[c][j] = v;
    }
}
// linear lateral test of one Gaussian against the views of zmask (set_lateral_bound in common.cuh): ALU only; the loop
// runs over the set bits (a depth candidate of a large scene is usually inside one view's depth range)
__device__ __forceinline__ uint32_t lateral_linear(const float (*s_lat)[kLatFloats], float px, float py, float pz, uint32_t zmask) {
    uint32_t keep = 0;
    while (zmask) {
        const int c = __ffs(zmask) - 1;
        zmask &= zmask - 1;
        const float* q = s_lat[c];
        const float tx = q[0] * px + q[1] * py + q[2] * pz + q[9];
        const float ty = q[3] * px + q[4] * py + q[5] * pz + q[10];
        const float tz = q[6] * px + q[7] * py + q[8] * pz + q[11];
        const bool out = (q[12] * fabsf(tx - tz * q[14]) > fmaf(q[16], tz, q[18])) || (q[13] * fabsf(ty - tz * q[15]) > fmaf(q[17], tz, q[18]));
        if (!out) keep |= 1u << c;
    }
    return keep;
}

// pop up to 32 entries from the top of `src` (one per lane), hand (index, mask, mean) of this lane's entry to `f`, which
// returns the new view mask; entries with a non-zero mask are pushed onto `dst`
template <typename Src, typename Dst, typename F>
__device__ __forceinline__ void stack_filter(Src& src, int& cnt_src, Dst& dst, int& cnt_dst, int lane, F f) {
    const int n = cnt_src < 32 ? cnt_src : 32;
    uint32_t idx[1] = {0u}, msk[1] = {0u};
    float m[3] = {0.f, 0.f, 0.f};
    if (lane < n) {
        const int p = cnt_src - n + lane;
        idx[0] = src.idx[p];
        m[0] = src.xyz[0][p]; m[1] = src.xyz[1][p]; m[2] = src.xyz[2][p];
        msk[0] = f(idx[0], src.msk[p], m);
    }
    cnt_src -= n;
    __syncwarp();      // the popped entries have been read
    warp_push<1>(idx, msk, m, dst, cnt_dst, lane);
    __syncwarp();
}

// Stages of a warp (each runs with full warps whenever 32 items are waiting, the later the stage the higher its priority;
// at the end of the input the stacks are drained):
//   A   streaming: means of a chunk -> near/far test of every view; zero radii / tiles_touched (or the mask words)  -> s1
//   B0a (only with the scene-wide scale bound) linear lateral test, ALU only                                        -> s1b
//   B0b the Gaussian's own largest scale (12-byte gather) -> conservative screen-space pre-cull                     -> s2
//   B1  full projection; SH only if visible somewhere
template <int DEG, int ITEMS>
__global__ void __launch_bounds__(kProjThreads, 6) project_fwd_kernel(const ProjFwdArgs a, const __grid_constant__ CamBatch cams) {
    pdl_enter();
    constexpr int CHUNK = 32 * ITEMS;                   // Gaussians per warp and phase-A step
    constexpr int WARPS = kProjThreads / 32;
    __shared__ WarpStack<32 + CHUNK, true> s1_all[WARPS];   // Gaussians inside some view's depth range
    __shared__ WarpStack<64, true> s1b_all[WARPS];          // ... that pass the linear lateral test with the scene-wide scale bound
    __shared__ WarpStack<64, true> s2_all[WARPS];           // survivors of the pre-cull with the Gaussian's own largest scale
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpStack<32 + CHUNK, true>& s1 = s1_all[warp];
    WarpStack<64, true>& s1b = s1b_all[warp];
    WarpStack<64, true>& s2 = s2_all[warp];
    const int64_t n_chunks = (a.N + CHUNK - 1) / CHUNK;
    const int64_t stride = (int64_t)gridDim.x * WARPS;
    int64_t chunk = (int64_t)blockIdx.x * WARPS + warp;
    int cnt1 = 0, cnt1b = 0, cnt2 = 0;    // warp-uniform stack heights
    float smax_all = -1.0f;
    if (a.ls_bound) smax_all = expf(__ldg(a.ls_bound));
    const bool use_bound = smax_all >= 0.0f && smax_all < kInfF;      // false for a NaN bound as well: nothing is dropped then
    __shared__ float s_lat[kMaxCamsPerLaunch][kLatFloats];
    if (use_bound) load_lateral_constants(cams, a.C, smax_all, s_lat);
    __syncthreads();       // (the only block barrier: from here on the warps run independently)
    while (true) {
        const bool more = chunk < n_chunks;
        if (cnt2 >= 32 || (cnt2 > 0 && !more && cnt1 == 0 && cnt1b == 0)) {
            // ---- B1: full projection of up to one survivor per lane
            const int n = cnt2 < 32 ? cnt2 : 32;
            if (lane < n) {
                const int p = cnt2 - n + lane;
                project_fwd_one<DEG>(a, cams, (int64_t)s2.idx[p], s2.msk[p], s2.xyz[0][p], s2.xyz[1][p], s2.xyz[2][p]);
            }
            cnt2 -= n;
            __syncwarp();          // the popped entries have been read
        } else if (cnt1b >= 32 || (cnt1b > 0 && !more && cnt1 == 0)) {
            // ---- B0b: screen-space pre-cull with the Gaussian's own largest scale -> s2
            stack_filter(s1b, cnt1b, s2, cnt2, lane, [&](uint32_t i, uint32_t zmask, const float* m) {
                const float* ls = a.log_scales + 3 * (int64_t)i;
                const float lmax = fmaxf(__ldg(ls), fmaxf(__ldg(ls + 1), __ldg(ls + 2)));
                return lateral_precull(a, cams, lmax, m[0], m[1], m[2], zmask);
            });
        } else if (cnt1 >= 32 || (cnt1 > 0 && !more)) {
            // ---- B0a: linear lateral test with the scene-wide bound (a plain move without one) -> s1b
            stack_filter(s1, cnt1, s1b, cnt1b, lane, [&](uint32_t, uint32_t zmask, const float* m) {
                return use_bound ? lateral_linear(s_lat, m[0], m[1], m[2], zmask) : zmask;
            });
        } else if (more) {
            // ---- A (streaming): means -> near/far test of every view; zero radii / tiles_touched (or the mask words) of the chunk
            const int64_t i0 = chunk * CHUNK + (int64_t)lane * ITEMS;
            float m[3 * ITEMS];
            const bool full = i0 + ITEMS <= a.N;
            if (ITEMS % 4 == 0 && a.vec_in && full) {
                const float4* p4 = reinterpret_cast<const float4*>(a.means + 3 * i0);
#pragma unroll
                for (int k = 0; k < 3 * ITEMS / 4; ++k) {
                    const float4 v = __ldg(p4 + k);
                    m[4 * k] = v.x; m[4 * k + 1] = v.y; m[4 * k + 2] = v.z; m[4 * k + 3] = v.w;
                }
            } else {
#pragma unroll
                for (int k = 0; k < 3 * ITEMS; ++k) m[k] = (i0 + k / 3 < a.N) ? __ldg(a.means + 3 * i0 + k) : 0.0f;
            }
            uint32_t idx[ITEMS], msk[ITEMS];
#pragma unroll
            for (int k = 0; k < ITEMS; ++k) msk[k] = 0;
            for (int c = 0; c < a.C; ++c) {
                const DevCam& cam = cams.cam[c];
                const float w0 = cam.W[6], w1 = cam.W[7], w2 = cam.W[8], t2 = cam.tau[2], zn = cam.near_plane, zf = cam.far_plane;
                const uint32_t bit = 1u << c;
                if (zn >= 0.0f && zf > zn) {
                    // zn < tz < zf on the bit patterns (non-negative floats order like their bits; a negative, zero or NaN tz wraps
                    // to or stays at a value above every range): one integer add and one unsigned compare per pair
                    const uint32_t lo = __float_as_uint(zn + 0.0f) + 1u, range = __float_as_uint(zf) - lo;
#pragma unroll
                    for (int k = 0; k < ITEMS; ++k) {
                        const float tz = w0 * m[3 * k] + w1 * m[3 * k + 1] + w2 * m[3 * k + 2] + t2;
                        msk[k] |= (__float_as_uint(tz) - lo < range) ? bit : 0u;
                    }
                } else {
#pragma unroll
                    for (int k = 0; k < ITEMS; ++k) {
                        const float tz = w0 * m[3 * k] + w1 * m[3 * k + 1] + w2 * m[3 * k + 2] + t2;
                        if (tz > zn && tz < zf) msk[k] |= bit;
                    }
                }
                const int64_t e0 = (int64_t)c * a.N + i0;
                if (a.vmask) {
                    // the chunk's ITEMS mask words of this view (and the row's padding words behind the last chunk)
                    uint32_t* row = a.vmask + (int64_t)c * a.wn;
                    if (lane < ITEMS) row[chunk * ITEMS + lane] = 0u;
                    if (chunk == n_chunks - 1 && n_chunks * ITEMS + lane < a.wn) row[n_chunks * ITEMS + lane] = 0u;
                } else if (ITEMS % 4 == 0 && a.vec_out && full) {
#pragma unroll
                    for (int k = 0; k < ITEMS / 4; ++k) {
                        reinterpret_cast<int4*>(a.radii + e0)[k] = make_int4(0, 0, 0, 0);
                        reinterpret_cast<uint4*>(a.tiles + e0)[k] = make_uint4(0u, 0u, 0u, 0u);
                    }
                } else {
#pragma unroll
                    for (int k = 0; k < ITEMS; ++k)
                        if (i0 + k < a.N) { a.radii[e0 + k] = 0; a.tiles[e0 + k] = 0u; }
                }
            }
#pragma unroll
            for (int k = 0; k < ITEMS; ++k) {
                if (i0 + k >= a.N) msk[k] = 0;
                idx[k] = (uint32_t)(i0 + k);
            }
            warp_push<ITEMS>(idx, msk, m, s1, cnt1, lane);
            chunk += stride;
            __syncwarp();      // pushes visible to the warp; its zero-fill is ordered before phase B's stores
        } else {
            break;
        }
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
    int32_t vec_in, vec_out;   // 16-byte vector access allowed on the radii rows / on the five gradient arrays
    int32_t prezeroed;         // the gradient arrays were zero-filled by zero_fill_kernel: phase A only reads the radii
    const uint32_t* vmask;     // optional visibility mask [C][wn] written by gs_project_fwd: read instead of the radii
    int64_t wn;
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

// phase B of P5 for one Gaussian visible in the views of `vis` (the rows were zero-filled in phase A
// unless the caller accumulates)
template <int DEG>
__device__ __forceinline__ void project_bwd_one(const ProjBwdArgs& a, const CamBatch& cams, int64_t i, uint32_t vis) {
    constexpr int K = (DEG + 1) * (DEG + 1);
    float gp[3] = {0.f, 0.f, 0.f}, gl[3] = {0.f, 0.f, 0.f}, gq[4] = {0.f, 0.f, 0.f, 0.f}, glogit = 0.f;
    float gsh[3 * K];
#pragma unroll
    for (int k = 0; k < 3 * K; ++k) gsh[k] = 0.f;

    {
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

// warp-cooperative zero-fill of `count` floats at p (16-byte stores when `vec`: p is then 16-byte aligned)
__device__ __forceinline__ void zero_span(float* __restrict__ p, int64_t count, bool vec, int lane) {
    if (vec) {
        const int64_t n4 = count >> 2;
        float4* p4 = reinterpret_cast<float4*>(p);
        for (int64_t k = lane; k < n4; k += 32) p4[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int64_t k = (n4 << 2) + lane; k < count; k += 32) p[k] = 0.f;
    } else {
        for (int64_t k = lane; k < count; k += 32) p[k] = 0.f;
    }
}

// MASK: visibility comes from the bit mask of gs_project_fwd; a lane then takes one mask word (32 Gaussians) per view,
// ITEMS = 32, and only the non-zero words are expanded (lane = bit).
template <int DEG, int ITEMS, bool MASK = false>
__global__ void __launch_bounds__(kBwdThreads, 3) project_bwd_kernel(const ProjBwdArgs a, const __grid_constant__ CamBatch cams) {
    pdl_enter();
    static_assert(!MASK || ITEMS == 32, "mask variant: one word per lane");
    constexpr int CHUNK = 32 * ITEMS;                   // Gaussians per warp and phase-A step
    constexpr int WARPS = kBwdThreads / 32;
    constexpr int K3 = 3 * (DEG + 1) * (DEG + 1);
    __shared__ WarpStack<32 + CHUNK, false> st_all[WARPS];   // visible Gaussians and the views they are visible in
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpStack<32 + CHUNK, false>& stk = st_all[warp];
    const int64_t n_chunks = (a.N + CHUNK - 1) / CHUNK;
    const int64_t stride = (int64_t)gridDim.x * WARPS;
    int64_t chunk = (int64_t)blockIdx.x * WARPS + warp;
    // MASK: a warp step takes 32 / kMaskGran granules of kMaskGran mask words that lie `stride` granules apart, i.e. consecutive
    // granules of the mask go to different warps: granule (kMaskGroups chunk' + q) * stride + g for the g-th warp, chunk' = 0,
    // 1, ... (`chunk` counts the warp's steps).  The visible Gaussians of a scene that is ordered in space (Morton order) sit
    // in a few index ranges; with 1 024 consecutive Gaussians per warp step a few hundred warps owned all of them, with
    // 256 per granule a range of 0.5 M Gaussians is spread over every resident warp.  Measured (P5 stage, ms; granule of
    // 32 / 16 / 8 words): city in Morton order 2.214 / 2.086 / 2.033, block 0.496 / 0.467 / 0.420; in generation order
    // city 2.121 / 2.128 / 2.143 (neighbouring visible Gaussians no longer share a warp round: their 236-byte rows are
    // gathered with less locality), block 0.434 / 0.433 / 0.434.  Prefetching the next step's words: slower (2.158).
    const int64_t gwarp = chunk;
    constexpr int kMaskGran = 8;                        // mask words per granule (8 words = one 32-byte sector = 256 Gaussians)
    constexpr int kMaskGroups = 32 / kMaskGran;         // granules per warp step
    const int64_t n_sectors = MASK ? a.wn / kMaskGran : 0;
    if constexpr (MASK) chunk = 0;
    int cnt = 0;               // warp-uniform stack height
    while (true) {
        // ---- phase A until a full warp of visible Gaussians is waiting: visibility from the saved
        //      radii; dense zero-fill of the chunk's gradient rows
        while (cnt < 32 && (MASK ? (kMaskGroups * chunk) * stride + gwarp < n_sectors : chunk < n_chunks)) {
            const int64_t base = chunk * CHUNK;
            const int64_t i0 = base + (int64_t)lane * ITEMS;
            if constexpr (MASK) {
                const int64_t word = ((kMaskGroups * chunk + lane / kMaskGran) * stride + gwarp) * kMaskGran + (lane % kMaskGran);   // this lane's word of every view's row
                uint32_t any = 0;
                if (word < a.wn)
                    for (int c = 0; c < a.C; ++c) any |= __ldg(a.vmask + (int64_t)c * a.wn + word);
                unsigned int nz = __ballot_sync(0xffffffffu, any != 0u);
                while (nz) {
                    const int sl = __ffs(nz) - 1;
                    nz &= nz - 1;
                    const int64_t ws = __shfl_sync(0xffffffffu, word, sl);
                    uint32_t idx1[1] = {(uint32_t)(ws * 32 + lane)}, vis1[1] = {0u};
                    for (int c = 0; c < a.C; ++c) vis1[0] |= ((__ldg(a.vmask + (int64_t)c * a.wn + ws) >> lane) & 1u) << c;   // (same address for all lanes)
                    warp_push<1>(idx1, vis1, nullptr, stk, cnt, lane);
                }
            } else {
            const bool full = i0 + ITEMS <= a.N;
            uint32_t idx[ITEMS], vis[ITEMS];
#pragma unroll
            for (int k = 0; k < ITEMS; ++k) vis[k] = 0;
            for (int c = 0; c < a.C; ++c) {
                const int64_t e0 = (int64_t)c * a.N + i0;
                if (ITEMS % 4 == 0 && a.vec_in && full) {
#pragma unroll
                    for (int q = 0; q < ITEMS / 4; ++q) {
                        const int4 r = __ldg(reinterpret_cast<const int4*>(a.radii + e0) + q);
                        vis[(4 * q) % ITEMS] |= (r.x > 0 ? 1u : 0u) << c; vis[(4 * q + 1) % ITEMS] |= (r.y > 0 ? 1u : 0u) << c;
                        vis[(4 * q + 2) % ITEMS] |= (r.z > 0 ? 1u : 0u) << c; vis[(4 * q + 3) % ITEMS] |= (r.w > 0 ? 1u : 0u) << c;
                    }
                } else {
#pragma unroll
                    for (int k = 0; k < ITEMS; ++k)
                        if (i0 + k < a.N && __ldg(a.radii + e0 + k) > 0) vis[k] |= 1u << c;
                }
            }
#pragma unroll
            for (int k = 0; k < ITEMS; ++k) idx[k] = (uint32_t)(i0 + k);
            warp_push<ITEMS>(idx, vis, nullptr, stk, cnt, lane);
            }
            if (!a.accumulate && !a.prezeroed) {
                const bool vec = a.vec_out != 0;
                // rows of this step: one span of CHUNK Gaussians, or (MASK) the 256 Gaussians of each of its four sectors
#pragma unroll 1
                for (int q = 0; q < (MASK ? kMaskGroups : 1); ++q) {
                    const int64_t zb = MASK ? ((kMaskGroups * chunk + q) * stride + gwarp) * (32 * kMaskGran) : base;
                    const int64_t span = MASK ? 32 * kMaskGran : CHUNK;
                    if (zb >= a.N) break;
                    const int64_t n = (a.N - zb) < span ? (a.N - zb) : span;
                    zero_span(a.d_sh + zb * K3, n * K3, vec, lane);
                    zero_span(a.d_means + zb * 3, n * 3, vec, lane);
                    zero_span(a.d_log_scales + zb * 3, n * 3, vec, lane);
                    zero_span(a.d_quats + zb * 4, n * 4, vec, lane);
                    zero_span(a.d_logits + zb, n, vec, lane);
                }
            }
            chunk += MASK ? 1 : stride;
            __syncwarp();      // pushes visible to the warp; its zero-fill is ordered before phase B's stores
        }
        // ---- phase B: gradients of up to one visible Gaussian per lane (top of the stack)
        if (cnt == 0) break;
        const int n = cnt < 32 ? cnt : 32;
        if (lane < n) project_bwd_one<DEG>(a, cams, (int64_t)stk.idx[cnt - n + lane], stk.msk[cnt - n + lane]);
        cnt -= n;
        __syncwarp();          // the popped entries have been read
    }
}

// Dense zero-fill of the five gradient arrays as one streaming kernel (16-byte stores, full occupancy).  For large N
// this is where P5's bytes go (236 B per Gaussian at SH degree 3); measured on B200 a plain store stream reaches
// 7.5 TB/s, the same stores issued from the 168-register persistent kernel's phase A 4.8 TB/s.
// one array: every thread zeroes four 16-byte units a block-width apart (coalesced, four stores in flight)
__global__ void __launch_bounds__(256) zero_fill_kernel(float* __restrict__ p, int64_t count) {
    pdl_enter();
    const int64_t n4 = count >> 2;
    const int64_t i0 = (int64_t)blockIdx.x * 1024 + threadIdx.x;
    float4* p4 = reinterpret_cast<float4*>(p);
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (i0 + k * 256 < n4) p4[i0 + k * 256] = zero;
    if (blockIdx.x == 0 && threadIdx.x < 4 && (n4 << 2) + threadIdx.x < count) p[(n4 << 2) + threadIdx.x] = 0.f;
}

// max over all log-scales (gs_log_scale_bound): 16-byte loads, warp shuffle, one atomic per warp
__global__ void __launch_bounds__(256) log_scale_max_kernel(const float* __restrict__ ls, int64_t n, int vec, float* __restrict__ out) {
    pdl_enter();
    float m = -3.0e38f;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x, t0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (vec) {
        const int64_t n4 = n >> 2;
        for (int64_t k = t0; k < n4; k += stride) {
            const float4 v = __ldg(reinterpret_cast<const float4*>(ls) + k);
            m = fmaxf(m, fmaxf(fmaxf(v.x, v.y), fmaxf(v.z, v.w)));
        }
        for (int64_t k = (n4 << 2) + t0; k < n; k += stride) m = fmaxf(m, __ldg(ls + k));
    } else {
        for (int64_t k = t0; k < n; k += stride) m = fmaxf(m, __ldg(ls + k));
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
    if ((threadIdx.x & 31) == 0 && m > -3.0e38f) {
        if (m >= 0.0f) atomicMax(reinterpret_cast<int*>(out), __float_as_int(m));
        else atomicMin(reinterpret_cast<unsigned int*>(out), __float_as_uint(m));
    }
}
__global__ void set_float_kernel(float* p, float v) { pdl_enter(); *p = v; }

// The same zero-fill as ONE launch with a small persistent grid (2 blocks of 256 threads per SM, 8 x 16-byte stores per
// thread and round): made to run on a second stream UNDERNEATH other kernels (gs_grad_zero_fill).  A full-size grid would
// take every free block slot of the SMs ahead of the kernels it is supposed to overlap with; two resident blocks per SM
// keep enough stores in flight for the full store bandwidth and leave the rest of the SM to the rasterisation kernels.
struct ZeroFillArgs {
    float* p[5];
    int64_t count[5];
};
__global__ void __launch_bounds__(256) zero_fill_persistent_kernel(const ZeroFillArgs a) {
    pdl_enter();
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    const int64_t stride = (int64_t)gridDim.x * 2048;
#pragma unroll 1
    for (int k = 0; k < 5; ++k) {
        float4* p4 = reinterpret_cast<float4*>(a.p[k]);
        const int64_t n4 = a.count[k] >> 2;
        for (int64_t i0 = (int64_t)blockIdx.x * 2048 + threadIdx.x; i0 < n4; i0 += stride) {
#pragma unroll
            for (int u = 0; u < 8; ++u)
                if (i0 + u * 256 < n4) p4[i0 + u * 256] = zero;
        }
        if (blockIdx.x == 0 && threadIdx.x < 4 && (n4 << 2) + threadIdx.x < a.count[k]) a.p[k][(n4 << 2) + threadIdx.x] = 0.f;
    }
}

// persistent grid: resident blocks of the kernel, or fewer when there are fewer chunks
template <typename Kernel>
static unsigned persistent_grid(Kernel kernel, int threads, int64_t n_chunks, int sms) {
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
    const int64_t resident = (int64_t)per_sm * sms;
    return (unsigned)(n_chunks < resident ? n_chunks : resident);
}

// several Gaussians per lane (16-byte accesses) when every resident warp still gets >= 8 chunks, else 1
template <int DEG>
int launch_fwd(const ProjFwdArgs& a, const CamBatch& cb, cudaStream_t st) {
    const int sms = sm_count();
    constexpr int warps = kProjThreads / 32;
    const int64_t wide = (a.N + 32 * kProjItems - 1) / (32 * kProjItems);
    const unsigned wide_grid = persistent_grid(project_fwd_kernel<DEG, kProjItems>, kProjThreads, (wide + warps - 1) / warps, sms);
    if (wide >= 8 * (int64_t)wide_grid * warps) {
        launch_chained(project_fwd_kernel<DEG, kProjItems>, dim3(wide_grid), dim3(kProjThreads), (size_t)(0), st, a, cb);
    } else {
        const int64_t chunks = (a.N + 31) / 32;
        launch_chained(project_fwd_kernel<DEG, 1>, dim3(persistent_grid(project_fwd_kernel<DEG, 1>, kProjThreads, (chunks + warps - 1) / warps, sms)), dim3(kProjThreads), (size_t)(0), st, a, cb);
    }
    return launch_status();
}
template <int DEG>
int launch_bwd(const ProjBwdArgs& a, const CamBatch& cb, cudaStream_t st) {
    const int sms = sm_count();
    constexpr int warps = kBwdThreads / 32;
    if (a.vmask) {
        const int64_t chunks = (a.N + 1023) / 1024;
        launch_chained(project_bwd_kernel<DEG, 32, true>, dim3(persistent_grid(project_bwd_kernel<DEG, 32, true>, kBwdThreads, (chunks + warps - 1) / warps, sms)), dim3(kBwdThreads), (size_t)(0), st, a, cb);
        return launch_status();
    }
    if (a.prezeroed || a.accumulate) {
        // phase A only scans the radii (or the visibility mask): 16 Gaussians per lane keep 4 C 16-byte loads in flight per lane
        // (only when every resident warp still gets >= 8 such chunks; else the narrower variants below)
        const int64_t scan = (a.N + 32 * 16 - 1) / (32 * 16);
        const unsigned scan_grid = persistent_grid(project_bwd_kernel<DEG, 16>, kBwdThreads, (scan + warps - 1) / warps, sms);
        if (scan >= 8 * (int64_t)scan_grid * warps) {
            launch_chained(project_bwd_kernel<DEG, 16>, dim3(scan_grid), dim3(kBwdThreads), (size_t)(0), st, a, cb);
            return launch_status();
        }
    }
    const int64_t wide = (a.N + 32 * 4 - 1) / (32 * 4);
    const unsigned wide_grid = persistent_grid(project_bwd_kernel<DEG, 4>, kBwdThreads, (wide + warps - 1) / warps, sms);
    if (wide >= 8 * (int64_t)wide_grid * warps) {
        launch_chained(project_bwd_kernel<DEG, 4>, dim3(wide_grid), dim3(kBwdThreads), (size_t)(0), st, a, cb);
    } else {
        const int64_t chunks = (a.N + 31) / 32;
        launch_chained(project_bwd_kernel<DEG, 1>, dim3(persistent_grid(project_bwd_kernel<DEG, 1>, kBwdThreads, (chunks + warps - 1) / warps, sms)), dim3(kBwdThreads), (size_t)(0), st, a, cb);
    }
    return launch_status();
}

}  // namespace gs

using namespace gs;

extern "C" int gs_project_fwd(const gs_config* cfg, int64_t N, const float* means, const float* log_scales,
                              const float* quats, const float* opacity_logits, const float* sh, int32_t C,
                              const gs_camera* cams, float* means2d, float* depths, float* conics, float* opacities,
                              float* rgbs, int32_t* radii, uint32_t* tiles_touched, uint32_t* vis_mask,
                              const float* log_scale_bound, void* stream) {
    int rc = check_cfg(cfg);
    if (rc) return rc;
    rc = check_cams(C, cams);
    if (rc) return rc;
    if (N < 0) return GS_ERR_INVALID_ARGUMENT;
    if (N == 0) return GS_OK;
    if (!means || !log_scales || !quats || !opacity_logits || !sh || !means2d || !depths || !conics || !opacities ||
        !rgbs || !radii || !tiles_touched)
        return GS_ERR_INVALID_ARGUMENT;
    if (!aligned(quats, 16) || !aligned(sh, 16) || !aligned(means2d, 8) || !aligned(means, 4) || !aligned(vis_mask, 16)) return GS_ERR_INVALID_ARGUMENT;
    if ((int64_t)C * N >= (1LL << 31)) return GS_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t wn = GS_VIS_WORDS(N);
    for (int c0 = 0; c0 < C; c0 += kMaxCamsPerLaunch) {
        const int nc = C - c0 < kMaxCamsPerLaunch ? C - c0 : kMaxCamsPerLaunch;
        CamBatch cb;
        for (int c = 0; c < nc; ++c) {
            cb.cam[c] = make_devcam(cams[c0 + c]);
            set_lateral_bound(cb.cam[c], cfg->extent, cfg->dilation);
        }
        ProjFwdArgs a;
        a.N = N; a.C = nc;
        a.means = means; a.log_scales = log_scales; a.quats = quats; a.logits = opacity_logits; a.sh = sh;
        const int64_t off = (int64_t)c0 * N;
        a.means2d = means2d + 2 * off; a.depths = depths + off; a.conics = conics + 3 * off;
        a.opacities = opacities + off; a.rgbs = rgbs + 3 * off; a.radii = radii + off; a.tiles = tiles_touched + off;
        a.dilation = cfg->dilation; a.extent = cfg->extent;
        a.vec_in = aligned(means, 16) ? 1 : 0;
        a.vec_out = (aligned(a.radii, 16) && aligned(a.tiles, 16) && (N % 4 == 0 || nc == 1)) ? 1 : 0;
        a.vmask = vis_mask ? vis_mask + (int64_t)c0 * wn : nullptr; a.wn = wn; a.ls_bound = log_scale_bound;
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

extern "C" int gs_log_scale_bound(int64_t N, const float* log_scales, float* bound, void* stream) {
    if (N < 1 || !log_scales || !bound || !aligned(bound, 4)) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t st = (cudaStream_t)stream;
    launch_chained(set_float_kernel, dim3(1), dim3(1), (size_t)(0), st, bound, -3.0e38f);
    const int64_t n = 3 * N;
    int64_t blocks = (n / 4 + 255) / 256;
    const int64_t cap = (int64_t)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    launch_chained(log_scale_max_kernel, dim3((unsigned)blocks), dim3(256), (size_t)(0), st, log_scales, n, aligned(log_scales, 16) ? 1 : 0, bound);
    return launch_status();
}

// dense zero-fill of the five gradient arrays (16-byte stores when the pointer allows it)
static int zero_fill_all(int64_t N, int sh_degree, float* dL_dmeans, float* dL_dlog_scales, float* dL_dquats, float* dL_dopacity_logits,
                         float* dL_dsh, cudaStream_t st) {
    const int64_t K3 = 3 * (int64_t)(sh_degree + 1) * (sh_degree + 1);
    float* ptrs[5] = {dL_dsh, dL_dquats, dL_dmeans, dL_dlog_scales, dL_dopacity_logits};
    const int64_t counts[5] = {K3 * N, 4 * N, 3 * N, 3 * N, N};
    for (int k = 0; k < 5; ++k) {
        if (aligned(ptrs[k], 16)) {
            const int64_t blocks = ((counts[k] >> 2) + 1023) / 1024;
            launch_chained(zero_fill_kernel, dim3((unsigned)(blocks > 0 ? blocks : 1)), dim3(256), (size_t)(0), st, ptrs[k], counts[k]);
        } else if (cudaMemsetAsync(ptrs[k], 0, (size_t)counts[k] * sizeof(float), st) != cudaSuccess) {
            return GS_ERR_CUDA;
        }
    }
    return launch_status();
}

extern "C" int gs_grad_zero_fill(int64_t N, int32_t sh_degree, float* dL_dmeans, float* dL_dlog_scales, float* dL_dquats,
                                 float* dL_dopacity_logits, float* dL_dsh, void* stream) {
    if (N < 0 || sh_degree < 0 || sh_degree > 3) return GS_ERR_INVALID_ARGUMENT;
    if (N == 0) return GS_OK;
    if (!dL_dmeans || !dL_dlog_scales || !dL_dquats || !dL_dopacity_logits || !dL_dsh) return GS_ERR_INVALID_ARGUMENT;
    if (aligned(dL_dmeans, 16) && aligned(dL_dlog_scales, 16) && aligned(dL_dquats, 16) && aligned(dL_dopacity_logits, 16) && aligned(dL_dsh, 16)) {
        const int64_t K3 = 3 * (int64_t)(sh_degree + 1) * (sh_degree + 1);
        ZeroFillArgs a;
        a.p[0] = dL_dsh; a.p[1] = dL_dquats; a.p[2] = dL_dmeans; a.p[3] = dL_dlog_scales; a.p[4] = dL_dopacity_logits;
        a.count[0] = K3 * N; a.count[1] = 4 * N; a.count[2] = 3 * N; a.count[3] = 3 * N; a.count[4] = N;
        launch_chained(zero_fill_persistent_kernel, dim3((unsigned)(2 * sm_count())), dim3(256), (size_t)(0), (cudaStream_t)stream, a);
        return launch_status();
    }
    return zero_fill_all(N, sh_degree, dL_dmeans, dL_dlog_scales, dL_dquats, dL_dopacity_logits, dL_dsh, (cudaStream_t)stream);
}

// Zero the rows of the Gaussians that a visibility mask marks in ANY of its C views (gs_grad_zero_rows).  A warp reads
// 32 consecutive mask words of every view (1024 Gaussians); every lane then clears the rows of the set bits of its own
// union word (a row is 236 contiguous-per-array bytes at SH degree 3: 12 + 1 16-byte stores and 7 scalar ones), so the
// rows of a chunk are cleared by up to 32 lanes at once.  City: 92 us for 0.59 M rows scattered over 14 GB (the same as a
// version that walked the rows one per warp round with the lanes sharing a row: the scattered partial-sector stores are
// the cost, not the instructions) against 1 870 us for the dense zero-fill.
struct ZeroRowsArgs {
    int64_t N, wn;
    int32_t C, K3, sh_vec, q_vec;
    const uint32_t* vmask;
    float* d_means; float* d_log_scales; float* d_quats; float* d_logits; float* d_sh;
};
__global__ void __launch_bounds__(256) zero_union_rows_kernel(const ZeroRowsArgs a) {
    pdl_enter();
    const int lane = threadIdx.x & 31;
    const int64_t n_chunks = (a.N + 1023) / 1024;
    const int64_t warps = (int64_t)gridDim.x * (blockDim.x >> 5);
    for (int64_t chunk = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); chunk < n_chunks; chunk += warps) {
        const int64_t w = chunk * 32 + lane;
        uint32_t u = 0;
        if (w < a.wn)
            for (int c = 0; c < a.C; ++c) u |= __ldg(a.vmask + (int64_t)c * a.wn + w);
        const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
        while (u) {
            const int64_t i = w * 32 + (__ffs(u) - 1);
            u &= u - 1;
            if (i >= a.N) break;
            if (a.sh_vec) {
                float4* p4 = reinterpret_cast<float4*>(a.d_sh + i * a.K3);
                for (int k = 0; k < a.K3 / 4; ++k) p4[k] = z4;
            } else {
                for (int k = 0; k < a.K3; ++k) a.d_sh[i * a.K3 + k] = 0.f;
            }
            if (a.q_vec) reinterpret_cast<float4*>(a.d_quats)[i] = z4;
            else { a.d_quats[4 * i] = 0.f; a.d_quats[4 * i + 1] = 0.f; a.d_quats[4 * i + 2] = 0.f; a.d_quats[4 * i + 3] = 0.f; }
            a.d_means[3 * i] = 0.f; a.d_means[3 * i + 1] = 0.f; a.d_means[3 * i + 2] = 0.f;
            a.d_log_scales[3 * i] = 0.f; a.d_log_scales[3 * i + 1] = 0.f; a.d_log_scales[3 * i + 2] = 0.f;
            a.d_logits[i] = 0.f;
        }
    }
}

extern "C" int gs_grad_zero_rows(int64_t N, int32_t sh_degree, int32_t C, const uint32_t* vis_mask, float* dL_dmeans, float* dL_dlog_scales,
                                 float* dL_dquats, float* dL_dopacity_logits, float* dL_dsh, void* stream) {
    if (N < 0 || sh_degree < 0 || sh_degree > 3 || C < 1 || C > GS_MAX_VIEWS) return GS_ERR_INVALID_ARGUMENT;
    if (N == 0) return GS_OK;
    if (!vis_mask || !aligned(vis_mask, 16) || !dL_dmeans || !dL_dlog_scales || !dL_dquats || !dL_dopacity_logits || !dL_dsh)
        return GS_ERR_INVALID_ARGUMENT;
    ZeroRowsArgs a;
    a.N = N; a.wn = GS_VIS_WORDS(N); a.C = C;
    a.K3 = 3 * (sh_degree + 1) * (sh_degree + 1);
    a.sh_vec = (a.K3 % 4 == 0 && aligned(dL_dsh, 16)) ? 1 : 0;
    a.q_vec = aligned(dL_dquats, 16) ? 1 : 0;
    a.vmask = vis_mask;
    a.d_means = dL_dmeans; a.d_log_scales = dL_dlog_scales; a.d_quats = dL_dquats; a.d_logits = dL_dopacity_logits; a.d_sh = dL_dsh;
    const int64_t chunks = (N + 1023) / 1024;
    const int64_t cap = (int64_t)sm_count() * 8;
    const int64_t blocks = (chunks + 7) / 8 < cap ? (chunks + 7) / 8 : cap;
    launch_chained(zero_union_rows_kernel, dim3((unsigned)blocks), dim3(256), (size_t)(0), (cudaStream_t)stream, a);
    return launch_status();
}

extern "C" int gs_project_bwd(const gs_config* cfg, int64_t N, const float* means, const float* log_scales,
                              const float* quats, const float* opacity_logits, const float* sh, int32_t C,
                              const gs_camera* cams, const int32_t* radii, const uint32_t* vis_mask, const float* dL_dmeans2d,
                              const float* dL_dconics, const float* dL_dopacities, const float* dL_drgbs,
                              float* dL_dmeans, float* dL_dlog_scales, float* dL_dquats, float* dL_dopacity_logits,
                              float* dL_dsh, int32_t accumulate, void* stream) {
    int rc = check_cfg(cfg);
    if (rc) return rc;
    rc = check_cams(C, cams);
    if (rc) return rc;
    if (N < 0) return GS_ERR_INVALID_ARGUMENT;
    if (N == 0) return GS_OK;
    if (!means || !log_scales || !quats || !opacity_logits || !sh || (!radii && !vis_mask) || !dL_dmeans2d || !dL_dconics ||
        !dL_dopacities || !dL_drgbs || !dL_dmeans || !dL_dlog_scales || !dL_dquats || !dL_dopacity_logits || !dL_dsh)
        return GS_ERR_INVALID_ARGUMENT;
    if (!aligned(quats, 16) || !aligned(sh, 16) || !aligned(dL_dquats, 16) || !aligned(dL_dsh, 16) || !aligned(dL_dmeans2d, 8))
        return GS_ERR_INVALID_ARGUMENT;
    if ((int64_t)C * N >= (1LL << 31)) return GS_ERR_UNSUPPORTED;
    if (accumulate < 0 || accumulate > 2) return GS_ERR_INVALID_ARGUMENT;
    if (accumulate == 2 && C > kMaxCamsPerLaunch) return GS_ERR_UNSUPPORTED;   // one launch must see every view of the batch
    cudaStream_t st = (cudaStream_t)stream;
    for (int c0 = 0; c0 < C; c0 += kMaxCamsPerLaunch) {
        const int nc = C - c0 < kMaxCamsPerLaunch ? C - c0 : kMaxCamsPerLaunch;
        CamBatch cb;
        for (int c = 0; c < nc; ++c) cb.cam[c] = make_devcam(cams[c0 + c]);
        ProjBwdArgs a;
        a.N = N; a.C = nc;
        a.means = means; a.log_scales = log_scales; a.quats = quats; a.logits = opacity_logits; a.sh = sh;
        const int64_t off = (int64_t)c0 * N;
        a.radii = radii ? radii + off : nullptr;
        a.vmask = vis_mask ? vis_mask + (int64_t)c0 * GS_VIS_WORDS(N) : nullptr; a.wn = GS_VIS_WORDS(N);
        a.g_means2d = dL_dmeans2d + 2 * off; a.g_conics = dL_dconics + 3 * off;
        a.g_opacities = dL_dopacities + off; a.g_rgbs = dL_drgbs + 3 * off;
        a.d_means = dL_dmeans; a.d_log_scales = dL_dlog_scales; a.d_quats = dL_dquats;
        a.d_logits = dL_dopacity_logits; a.d_sh = dL_dsh;
        a.dilation = cfg->dilation;
        // the first chunk of cameras overwrites (unless the caller accumulates), later chunks add
        // accumulate == 2 ("visible rows only"): the rows of Gaussians visible in this batch are overwritten, all other rows
        // are left untouched (no dense zero-fill: the caller's optimizer reads only visible rows, gs_adam_step_visible)
        a.accumulate = (accumulate == 1 || c0 > 0) ? 1 : 0;
        a.vec_in = (a.radii && aligned(a.radii, 16) && (N % 4 == 0 || nc == 1)) ? 1 : 0;
        a.vec_out = (aligned(dL_dmeans, 16) && aligned(dL_dlog_scales, 16) && aligned(dL_dquats, 16) &&
                     aligned(dL_dopacity_logits, 16) && aligned(dL_dsh, 16)) ? 1 : 0;
        a.prezeroed = (accumulate == 2) ? 1 : 0;
        if (!a.accumulate && accumulate != 2 && a.vec_out && N >= kZeroFillMinN) {
            rc = zero_fill_all(N, cfg->sh_degree, dL_dmeans, dL_dlog_scales, dL_dquats, dL_dopacity_logits, dL_dsh, st);
            if (rc) return rc;
            a.prezeroed = 1;
        }
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
