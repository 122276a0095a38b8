// raster.cu -- per-pixel stages R1 (gs_raster_fwd) and R2 (gs_raster_bwd) plus the harness L1 loss.
//
// One 128-thread block per (view, tile); each of its 4 warps owns an 8x8 pixel block of the 16x16
// tile and every lane two horizontally adjacent pixels, evaluated together with the two-wide FP32
// instructions of sm_100a (FFMA2 / FMUL2 / FADD2): both kernels are issue bound, and one packed
// instruction takes one issue slot for two pixels.  The tile's sorted records are staged through
// shared memory in batches (one gathered record per thread, conic pre-scaled to the log2 domain,
// every field stored twice so that one LDS.128 yields two operand pairs).  Only ~1/4 of the (pixel,
// record) pairs of a tile list pass the alpha >= alpha_min rule, so before evaluating anything a
// warp FILTERS the batch: lane l bounds record (chunk*32 + l) over the warp's 8x8 pixel rectangle
// (exact maximum of the concave exponent over the rectangle, conservative margin) and a ballot
// gives the records that can contribute; the warp then walks only those bits.  The filter never
// changes a per-pixel decision, it only skips records for which every pixel would be skipped.
// Forward: a warp stops when all its pixels are saturated, the block stops fetching when every warp
// has.  Backward: back to front from the tile's largest n_contrib; per (pixel,
// record) pair only dL/dpower and alpha*T are produced, transposed through a shared-memory tile
// and contracted with the pixel offsets (moments) by the lanes of the record; the 9 sums of a
// record go to the warp's own shared-memory slot (shared-memory float atomics are CAS loops on
// this hardware), are summed across the 4 warps at the end of the batch and flushed with one
// device-scope red.add per value and (tile, record).
#include "common.cuh"

namespace gs {

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kFilterMargin = 0.01f;  // log2 units: a record is dropped only if alpha < 0.993 alpha_min everywhere

struct RasterArgs {
    int32_t width, height, gx, gy;
    int64_t tiles;
    const int32_t* vals; const int64_t* ranges;
    const float* means2d; const float* conics; const float* opacities; const float* rgbs;
    float bg0, bg1, bg2;
    float alpha_min, alpha_max, t_min;
    float filter_thr;      // log2(alpha_min) - margin (-inf when alpha_min <= 0)
};

struct RasterFwdOut {
    float* image; float* final_T; int32_t* n_contrib;
};

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// scaled exponent e(dx,dy) = A' dx^2 + B' dx dy + C' dy^2  (= power * log2(e))
__device__ __forceinline__ float quad_form(float A, float B, float C, float dx, float dy) {
    const float t = fmaf(B, dy, A * dx);
    return fmaf(C * dy, dy, t * dx);
}

// position of the most significant set bit (x != 0)
__device__ __forceinline__ int msb(unsigned int x) {
    int r;
    asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(x));
    return r;
}
__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
// ---- packed FP32 (two pixels per lane) ---------------------------------------------------------
// sm_100a has two-wide FP32 instructions (FFMA2 / FMUL2 / FADD2 on 64-bit register pairs; PTX
// fma/mul/add.rn.f32x2).  The raster kernels are issue bound, so a lane owns two horizontally
// adjacent pixels and evaluates the exponent, the transmittance update and the colour sums of both
// with one instruction each.  Records are staged with every field duplicated so that one LDS.128
// yields two ready-made operand pairs.
__device__ __forceinline__ void lds2x64(uint32_t addr, f32x2& a, f32x2& b) {
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "r"(addr));
}
__device__ __forceinline__ f32x2 lds64(uint32_t addr) {
    f32x2 a;
    asm volatile("ld.shared.b64 %0, [%1];" : "=l"(a) : "r"(addr));
    return a;
}

// One staged record of the packed kernels: 80 bytes, every operand of the per-pixel arithmetic twice.
struct __align__(16) Rec {
    float4 a;   // u, u, v, v
    float4 b;   // A', A', B', B'
    float4 c;   // C', C', log2(opacity) x 2
    float4 d;   // r, r, g, g
    float4 e;   // b, b, bit pattern of the entry id, opacity
};

__device__ __forceinline__ void stage_record(const RasterArgs& a, int g, Rec& r) {
    const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + g);
    const float A = -0.5f * kLog2e * __ldg(a.conics + 3 * (int64_t)g), B = -kLog2e * __ldg(a.conics + 3 * (int64_t)g + 1),
                Cc = -0.5f * kLog2e * __ldg(a.conics + 3 * (int64_t)g + 2);
    const float op = __ldg(a.opacities + g);
    const float lo = __log2f(op);
    const float cr = __ldg(a.rgbs + 3 * (int64_t)g), cg = __ldg(a.rgbs + 3 * (int64_t)g + 1), cb = __ldg(a.rgbs + 3 * (int64_t)g + 2);
    r.a = make_float4(uv.x, uv.x, uv.y, uv.y);
    r.b = make_float4(A, A, B, B);
    r.c = make_float4(Cc, Cc, lo, lo);
    r.d = make_float4(cr, cr, cg, cg);
    r.e = make_float4(cb, cb, __int_as_float(g), op);
}

// rect_may_contribute for a (wx+1) x (wy+1) block of pixel centres starting at (X0, Y0)
__device__ __forceinline__ bool rect_may_contribute(float u, float v, float A, float B, float C, float lo, float X0, float Y0, float wx, float wy,
                                                     float thr) {
    const float dx0 = u - (X0 + wx), dx1 = u - X0;
    const float dy0 = v - (Y0 + wy), dy1 = v - Y0;
    const bool inx = (dx0 <= 0.0f) && (dx1 >= 0.0f), iny = (dy0 <= 0.0f) && (dy1 >= 0.0f);
    const bool concave = (A <= 0.0f) && (C <= 0.0f) && (4.0f * A * C - B * B >= 0.0f);
    float emax = 0.0f;
    if (!(inx && iny)) {
        emax = -3.0e38f;
        if (!inx) {
            const float dxe = dx0 > 0.0f ? dx0 : dx1;
            const float dys = fminf(fmaxf(-0.5f * B * dxe * rcp_approx(C), dy0), dy1);
            emax = fmaxf(emax, fmaxf(quad_form(A, B, C, dxe, dys), fmaxf(quad_form(A, B, C, dxe, dy0), quad_form(A, B, C, dxe, dy1))));
        }
        if (!iny) {
            const float dye = dy0 > 0.0f ? dy0 : dy1;
            const float dxs = fminf(fmaxf(-0.5f * B * dye * rcp_approx(A), dx0), dx1);
            emax = fmaxf(emax, fmaxf(quad_form(A, B, C, dxs, dye), fmaxf(quad_form(A, B, C, dx0, dye), quad_form(A, B, C, dx1, dye))));
        }
    }
    return !concave || !(emax + lo < thr);
}

constexpr int kBlock = 128;    // 4 warps per tile, each an 8x8 pixel block, lane = 2 x 1 pixels

__global__ void __launch_bounds__(kBlock) raster_fwd_kernel(const RasterArgs a, const RasterFwdOut o) {
    pdl_enter();
    __shared__ Rec s_rec[kBlock];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t bt = blockIdx.x;                  // view * tiles + tile
    const int64_t view = bt / a.tiles;
    const int t = (int)(bt - view * a.tiles);
    const int ty = t / a.gx, tx = t - ty * a.gx;
    const int bx0 = tx * kTile + (warp & 1) * 8, by0 = ty * kTile + (warp >> 1) * 8;   // the warp's 8x8 pixel block
    const int j = bx0 + 2 * (lane & 3), i = by0 + (lane >> 2);                          // pixels (i, j) and (i, j + 1)
    const bool in0 = (i < a.height) && (j < a.width), in1 = (i < a.height) && (j + 1 < a.width);
    const f32x2 npx = pk2(-((float)j + 0.5f), -((float)j + 1.5f));
    const float npy_s = -((float)i + 0.5f);
    const f32x2 npy = pk2(npy_s, npy_s);
    const f32x2 one2 = pk2(1.0f, 1.0f), neg2 = pk2(-1.0f, -1.0f);
    const float X0 = (float)bx0 + 0.5f, Y0 = (float)by0 + 0.5f;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(s_rec);
    const float alpha_min = a.alpha_min, alpha_max = a.alpha_max, t_min = a.t_min;

    const int64_t start = __ldg(a.ranges + 2 * bt), end = __ldg(a.ranges + 2 * bt + 1);
    // A pixel that has terminated (or lies outside the image) carries its transmittance NEGATED: T (1 - alpha) is then
    // negative, fails the T' >= t_min test and nothing updates any more -- the sticky "done" flag costs no predicate
    // register and no select of its own (the ALU pipe, half as wide as the FMA pipe, is the busiest unit of this loop).
    float T0 = in0 ? 1.0f : -1.0f, T1 = in1 ? 1.0f : -1.0f;
    f32x2 c0 = pk2(0.f, 0.f), c1 = c0, c2 = c0;
    int last0 = 0, last1 = 0;
    for (int64_t base = start; base < end; base += kBlock) {
        if (__syncthreads_and(T0 < 0.0f && T1 < 0.0f)) break;
        const int64_t k = base + tid;
        if (k < end) stage_record(a, __ldg(a.vals + k), s_rec[tid]);
        __syncthreads();
        const int cnt = (int)((end - base) < kBlock ? (end - base) : kBlock);
        const int nbase = (int)(base - start) + 1;
        bool warp_done = __all_sync(0xffffffffu, T0 < 0.0f && T1 < 0.0f);
        for (int ch = 0; ch * 32 < cnt && !warp_done; ++ch) {
            const int r = ch * 32 + lane;
            bool may = false;
            if (r < cnt) {
                const Rec& rc = s_rec[r];
                may = rect_may_contribute(rc.a.x, rc.a.z, rc.b.x, rc.b.z, rc.c.x, rc.c.z, X0, Y0, 7.0f, 7.0f, a.filter_thr);
            }
            unsigned int mask = __ballot_sync(0xffffffffu, may);
            // (Round 1 dropped the "power > 0" test for chunks of concave conics; the backward kernel always applies it, and for
            //  near-singular conics the fp32 exponent is +-1e-4 around 0, so the two passes disagreed on such pairs.  Always
            //  applying it, as O-R1 is written, costs 2 % here; the same per-chunk rule in the backward kernel cost it 1-4 %.)
            while (mask) {
                const int q = ch * 32 + __ffs(mask) - 1;
                mask &= mask - 1;
                const uint32_t addr = sbase + (uint32_t)q * (uint32_t)sizeof(Rec);
                f32x2 uu, vv, AA, BB, CC, LL, rr, gg;
                lds2x64(addr, uu, vv);
                lds2x64(addr + 16, AA, BB);
                lds2x64(addr + 32, CC, LL);
                lds2x64(addr + 48, rr, gg);
                const f32x2 bb = lds64(addr + 64);
                const f32x2 dx = add2(uu, npx), dy = add2(vv, npy);
                // same operation order as quad_form: t = fma(B, dy, A dx); e = fma(C dy, dy, t dx)
                const f32x2 tq = fma2(BB, dy, mul2(AA, dx));
                const f32x2 e2 = fma2(mul2(CC, dy), dy, mul2(tq, dx));
                const f32x2 el = add2(e2, LL);
                float e_0, e_1, el0, el1;
                unpk2(e2, e_0, e_1);
                unpk2(el, el0, el1);
                const float al0 = fminf(alpha_max, ex2_approx(el0)), al1 = fminf(alpha_max, ex2_approx(el1));
                const f32x2 al = pk2(al0, al1), Tp = pk2(T0, T1);
                const f32x2 Tn = mul2(Tp, fma2(al, neg2, one2));      // T (1 - alpha)
                const f32x2 wg = mul2(al, Tp);
                float Tn0, Tn1, wg0, wg1;
                unpk2(Tn, Tn0, Tn1);
                unpk2(wg, wg0, wg1);
                const bool ok0 = !(e_0 > 0.0f) && !(al0 < alpha_min), ok1 = !(e_1 > 0.0f) && !(al1 < alpha_min);
                const bool term0 = ok0 && (Tn0 < t_min), term1 = ok1 && (Tn1 < t_min);      // also true again for a finished pixel
                const bool upd0 = ok0 && !(Tn0 < t_min), upd1 = ok1 && !(Tn1 < t_min);
                const f32x2 w2 = pk2(upd0 ? wg0 : 0.0f, upd1 ? wg1 : 0.0f);
                c0 = fma2(rr, w2, c0);
                c1 = fma2(gg, w2, c1);
                c2 = fma2(bb, w2, c2);
                T0 = upd0 ? Tn0 : (term0 ? -fabsf(T0) : T0);
                T1 = upd1 ? Tn1 : (term1 ? -fabsf(T1) : T1);
                last0 = upd0 ? nbase + q : last0; last1 = upd1 ? nbase + q : last1;
                if (__all_sync(0xffffffffu, T0 < 0.0f && T1 < 0.0f)) { warp_done = true; break; }
            }
        }
    }
    float r0, r1, g0, g1, b0, b1;
    unpk2(c0, r0, r1); unpk2(c1, g0, g1); unpk2(c2, b0, b1);
    const int64_t pix = (view * a.height + i) * a.width + j;
    T0 = fabsf(T0); T1 = fabsf(T1);
    if (in0) {
        o.image[3 * pix] = r0 + T0 * a.bg0; o.image[3 * pix + 1] = g0 + T0 * a.bg1; o.image[3 * pix + 2] = b0 + T0 * a.bg2;
        o.final_T[pix] = T0;
        o.n_contrib[pix] = last0;
    }
    if (in1) {
        o.image[3 * pix + 3] = r1 + T1 * a.bg0; o.image[3 * pix + 4] = g1 + T1 * a.bg1; o.image[3 * pix + 5] = b1 + T1 * a.bg2;
        o.final_T[pix + 1] = T1;
        o.n_contrib[pix + 1] = last1;
    }
}

// ---------------------------------------------------------------------------------------------
struct RasterBwdIO {
    const float* final_T; const int32_t* n_contrib; const float* dL_dimage;
    float* g_means2d; float* g_conics; float* g_opacities; float* g_rgbs;
};

// ---- backward ------------------------------------------------------------------------------------
// Per (pixel, record) pair the backward pass produces two scalars: gp = dL/dpower and wgt = alpha*T
// (the weight of dL/dimage in dL/drgb).  Every per-record sum is a contraction of those over the
// pixels: with pixel offsets (x, y) from the tile centre, the geometric gradients need the moments
// sum gp*{1, x, y, x^2, xy, y^2} and dL/drgb needs sum wgt*g_c -- 9 values.  Instead of a 32-lane
// butterfly per record, a warp TRANSPOSES: lane = pixel pair writes (gp, wgt) of up to 8 records
// into a shared-memory tile, then lane (record g, row pair t) reads its 16 pixels (LDS.128),
// accumulates the moments with immediate x offsets (FFMA), and only the 4 lanes of a record are
// combined by shuffles (value-splitting, 8 shuffles per 8 records).
// 4 warps per tile, each an 8x8 pixel block (lane = row l >> 2, columns 2 (l & 3) and
// 2 (l & 3) + 1).  Transposition tile: one row per
// record, 64 pixels in row-major order of the 8x8 block, 4 floats of padding after pixel 31 and a
// row stride of 72 floats, so that both the 64-bit stores of the evaluation phase and the 128-bit
// loads of the reduction phase (lane (record g, row pair t) reads pixels 16 t .. 16 t + 15) are free
// of bank conflicts.
constexpr int kBwdBatch = 64;
constexpr int kBwdChunks = kBwdBatch / 32;
constexpr int kWarps = kBlock / 32;
constexpr int kTStride = 72;                // floats per transposition row: 64 pixels + 4 + 4
constexpr int kGroup = 8;                   // records reduced together by one warp
constexpr int kSlot = 9;                    // floats per (warp, record) slot (odd stride: conflict-free flush)

struct BwdSmem {
    Rec rec[kBwdBatch];
    float slot[kWarps][kBwdBatch][kSlot];     // m0, m1x, m1y, m2xx, m2xy, m2yy, dr, dg, (db at [8])
    float tbuf[kWarps][2 * kGroup][kTStride]; // rows 0..7: gp of record k over the warp's 64 pixels; rows 8..15: wgt
    float gpix[kWarps][3][kTStride];          // dL/dimage of the warp's pixels, one row per channel, same pixel layout
    unsigned int vis[kWarps][kBwdChunks];
    int max_contrib;
};

__device__ __forceinline__ void sts64(uint32_t addr, f32x2 v) { asm volatile("st.shared.b64 [%0], %1;" :: "r"(addr), "l"(v)); }

// moments of one row of 8 values about the centre of the 8 columns (x = -3.5 .. 3.5)
__device__ __forceinline__ void row_moments(const float4 p0, const float4 p1, float& s0, float& s1, float& s2) {
    const float a0 = p0.x + p1.w, a1 = p0.y + p1.z, a2 = p0.z + p1.y, a3 = p0.w + p1.x;
    const float d0 = p1.w - p0.x, d1 = p1.z - p0.y, d2 = p1.y - p0.z, d3 = p1.x - p0.w;
    s0 = (a0 + a1) + (a2 + a3);
    s1 = fmaf(3.5f, d0, fmaf(2.5f, d1, fmaf(1.5f, d2, 0.5f * d3)));
    s2 = fmaf(12.25f, a0, fmaf(6.25f, a1, fmaf(2.25f, a2, 0.25f * a3)));
}
__device__ __forceinline__ float dot8(const float4 w0, const float4 w1, const float4 g0, const float4 g1, float acc) {
    acc = fmaf(w0.x, g0.x, acc); acc = fmaf(w0.y, g0.y, acc); acc = fmaf(w0.z, g0.z, acc); acc = fmaf(w0.w, g0.w, acc);
    acc = fmaf(w1.x, g1.x, acc); acc = fmaf(w1.y, g1.y, acc); acc = fmaf(w1.z, g1.z, acc); acc = fmaf(w1.w, g1.w, acc);
    return acc;
}

// Reduce the k (<= 8) records of a warp's group.  lane = 4 g + t: record g, pixel rows 2 t and 2 t + 1
// of the warp's block; `pya` = offset of row 2 t from the tile centre, `ox` = offset of the centre of
// the warp's 8 columns; `myq` = batch position of record g.
__device__ __forceinline__ void reduce_group(BwdSmem& sm, int warp, int lane, int k, int myq, float ox, float pya) {
    __syncwarp();
    const int g = lane >> 2, t = lane & 3;
    const int poff = 16 * t + ((t >> 1) << 2);
    const uint32_t tb = (uint32_t)__cvta_generic_to_shared(&sm.tbuf[warp][g][poff]);
    const uint32_t wb = tb + kGroup * kTStride * 4;
    const uint32_t gb = (uint32_t)__cvta_generic_to_shared(&sm.gpix[warp][0][poff]);
    const float pyb = pya + 1.0f;
    float s0a, s1a, s2a, s0b, s1b, s2b;
    row_moments(lds128(tb), lds128(tb + 16), s0a, s1a, s2a);
    row_moments(lds128(tb + 32), lds128(tb + 48), s0b, s1b, s2b);
    float v[9];
    const float s0 = s0a + s0b, s1 = s1a + s1b, s2 = s2a + s2b;
    const float m1xa = fmaf(ox, s0a, s1a), m1xb = fmaf(ox, s0b, s1b);
    const float m1x = m1xa + m1xb;
    const float ya = pya * s0a, yb = pyb * s0b;
    v[0] = s0;
    v[1] = m1x;
    v[2] = ya + yb;
    v[3] = fmaf(ox, m1x + s1, s2);            // s2 + 2 ox s1 + ox^2 s0
    v[4] = fmaf(pya, m1xa, pyb * m1xb);
    v[5] = fmaf(pya, ya, pyb * yb);
    const float4 w0 = lds128(wb), w1 = lds128(wb + 16), w2 = lds128(wb + 32), w3 = lds128(wb + 48);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const uint32_t ga = gb + c * kTStride * 4;
        float acc = dot8(w0, w1, lds128(ga), lds128(ga + 16), 0.0f);
        v[6 + c] = dot8(w2, w3, lds128(ga + 32), lds128(ga + 48), acc);
    }
    // combine the 4 lanes of a record: values 0..7 split, value 8 plain
    const bool b1 = t & 2, b0 = t & 1;
    float c0, c1, c2, c3;
    {
        const float s_0 = b1 ? v[0] : v[4], s_1 = b1 ? v[1] : v[5], s_2 = b1 ? v[2] : v[6], s_3 = b1 ? v[3] : v[7];
        const float k_0 = b1 ? v[4] : v[0], k_1 = b1 ? v[5] : v[1], k_2 = b1 ? v[6] : v[2], k_3 = b1 ? v[7] : v[3];
        c0 = k_0 + __shfl_xor_sync(0xffffffffu, s_0, 2);
        c1 = k_1 + __shfl_xor_sync(0xffffffffu, s_1, 2);
        c2 = k_2 + __shfl_xor_sync(0xffffffffu, s_2, 2);
        c3 = k_3 + __shfl_xor_sync(0xffffffffu, s_3, 2);
    }
    float e0, e1;
    {
        const float s_0 = b0 ? c0 : c2, s_1 = b0 ? c1 : c3;
        const float k_0 = b0 ? c2 : c0, k_1 = b0 ? c3 : c1;
        e0 = k_0 + __shfl_xor_sync(0xffffffffu, s_0, 1);
        e1 = k_1 + __shfl_xor_sync(0xffffffffu, s_1, 1);
    }
    float w = v[8];
    w += __shfl_xor_sync(0xffffffffu, w, 2);
    w += __shfl_xor_sync(0xffffffffu, w, 1);
    if (g < k) {
        float* slot = &sm.slot[warp][myq][0];
        slot[2 * t] = e0;
        slot[2 * t + 1] = e1;
        if (t == 0) slot[8] = w;
    }
    __syncwarp();
}

__global__ void __launch_bounds__(kBlock) raster_bwd_kernel(const RasterArgs a, const RasterBwdIO io) {
    pdl_enter();
    extern __shared__ __align__(16) unsigned char bwd_smem_raw[];
    BwdSmem& sm = *reinterpret_cast<BwdSmem*>(bwd_smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t bt = blockIdx.x;
    const int64_t view = bt / a.tiles;
    const int t = (int)(bt - view * a.tiles);
    const int ty = t / a.gx, tx = t - ty * a.gx;
    const int bx0 = tx * kTile + (warp & 1) * 8, by0 = ty * kTile + (warp >> 1) * 8;
    const int j = bx0 + 2 * (lane & 3), i = by0 + (lane >> 2);
    const bool in0 = (i < a.height) && (j < a.width), in1 = (i < a.height) && (j + 1 < a.width);
    const f32x2 npx = pk2(-((float)j + 0.5f), -((float)j + 1.5f));
    const float npy_s = -((float)i + 0.5f);
    const f32x2 npy = pk2(npy_s, npy_s);
    const f32x2 one2 = pk2(1.0f, 1.0f), neg2 = pk2(-1.0f, -1.0f);
    const float X0 = (float)bx0 + 0.5f, Y0 = (float)by0 + 0.5f;
    const float xc = (float)(tx * kTile + kTile / 2), yc = (float)(ty * kTile + kTile / 2);   // tile centre
    const float ox = (warp & 1) ? 4.0f : -4.0f;                                            // centre of the warp's columns - xc
    const float pya = (float)((warp >> 1) * 8 + 2 * (lane & 3)) + 0.5f - 8.0f;             // reduce-phase row 2 (lane & 3) - yc
    const int64_t start = __ldg(a.ranges + 2 * bt);
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(sm.rec);
    const int ppos = 2 * lane + ((lane >> 4) << 2);                                        // this lane's pixel pair in a tile row
    const uint32_t tbase = (uint32_t)__cvta_generic_to_shared(&sm.tbuf[warp][0][ppos]);
    const float alpha_min = a.alpha_min, alpha_max = a.alpha_max;

    float T0 = 0.f, T1 = 0.f;
    float gr0 = 0.f, gg0 = 0.f, gb0 = 0.f, gr1 = 0.f, gg1 = 0.f, gb1 = 0.f;
    int ncon0 = 0, ncon1 = 0;
    const int64_t pix = (view * a.height + i) * a.width + j;
    if (in0) {
        T0 = __ldg(io.final_T + pix);
        ncon0 = __ldg(io.n_contrib + pix);
        gr0 = __ldg(io.dL_dimage + 3 * pix); gg0 = __ldg(io.dL_dimage + 3 * pix + 1); gb0 = __ldg(io.dL_dimage + 3 * pix + 2);
    }
    if (in1) {
        T1 = __ldg(io.final_T + pix + 1);
        ncon1 = __ldg(io.n_contrib + pix + 1);
        gr1 = __ldg(io.dL_dimage + 3 * pix + 3); gg1 = __ldg(io.dL_dimage + 3 * pix + 4); gb1 = __ldg(io.dL_dimage + 3 * pix + 5);
    }
    {
        float* gp = &sm.gpix[warp][0][ppos];
        gp[0] = gr0; gp[1] = gr1;
        gp[kTStride] = gg0; gp[kTStride + 1] = gg1;
        gp[2 * kTStride] = gb0; gp[2 * kTStride + 1] = gb1;
    }
    const f32x2 G0 = pk2(gr0, gr1), G1 = pk2(gg0, gg1), G2 = pk2(gb0, gb1);
    if (tid == 0) sm.max_contrib = 0;
    __syncthreads();
    int wmax = max(ncon0, ncon1);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, d));
    if (lane == 0 && wmax > 0) atomicMax(&sm.max_contrib, wmax);
    __syncthreads();
    const int maxn = sm.max_contrib;
    if (maxn == 0) return;
    // colour accumulated behind the current record
    f32x2 S0 = pk2(a.bg0, a.bg0), S1 = pk2(a.bg1, a.bg1), S2 = pk2(a.bg2, a.bg2);
    const int nb = (maxn + kBwdBatch - 1) / kBwdBatch;
    for (int b = nb - 1; b >= 0; --b) {
        const int cnt = min(kBwdBatch, maxn - b * kBwdBatch);
        __syncthreads();   // previous batch fully flushed
        if (tid < cnt) stage_record(a, __ldg(a.vals + start + (int64_t)b * kBwdBatch + tid), sm.rec[tid]);
        __syncthreads();
        int k = 0;         // records in the warp's current group (warp-uniform)
        int myq = 0;       // batch position of the group's record (lane >> 2)
        uint32_t taddr = tbase;   // this lane's cell in row k of the transposition tile
        for (int ch = kBwdChunks - 1; ch >= 0; --ch) {
            const int r = ch * 32 + lane;
            const int cbase = b * kBwdBatch + ch * 32;         // list position of bit 0 of this chunk
            bool may = false;
            if (r < cnt && (cbase + lane) < wmax) {
                const Rec& rc = sm.rec[r];
                may = rect_may_contribute(rc.a.x, rc.a.z, rc.b.x, rc.b.z, rc.c.x, rc.c.z, X0, Y0, 7.0f, 7.0f, a.filter_thr);
            }
            unsigned int mask = __ballot_sync(0xffffffffu, may);
            const int nrel0 = ncon0 - cbase, nrel1 = ncon1 - cbase;   // pixel j walks bits < nrel_j
            unsigned int written = 0;
            const uint32_t cbase_addr = sbase + (uint32_t)(ch * 32) * (uint32_t)sizeof(Rec);
            while (mask) {
                const int bit = msb(mask);
                mask ^= 1u << bit;
                const uint32_t addr = cbase_addr + (uint32_t)bit * (uint32_t)sizeof(Rec);
                f32x2 uu, vv, AA, BB, CC, LL;
                lds2x64(addr, uu, vv);
                lds2x64(addr + 16, AA, BB);
                lds2x64(addr + 32, CC, LL);
                const f32x2 dx = add2(uu, npx), dy = add2(vv, npy);
                const f32x2 tq = fma2(BB, dy, mul2(AA, dx));
                const f32x2 e2 = fma2(mul2(CC, dy), dy, mul2(tq, dx));
                const f32x2 el = add2(e2, LL);
                float e_0, e_1, el0, el1;
                unpk2(e2, e_0, e_1);
                unpk2(el, el0, el1);
                const float raw0 = ex2_approx(el0), raw1 = ex2_approx(el1);
                const float al0 = fminf(alpha_max, raw0), al1 = fminf(alpha_max, raw1);
                const bool valid0 = (bit < nrel0) && !(e_0 > 0.0f) && !(al0 < alpha_min);
                const bool valid1 = (bit < nrel1) && !(e_1 > 0.0f) && !(al1 < alpha_min);
                if (!__any_sync(0xffffffffu, valid0 || valid1)) continue;
                f32x2 rr, gg;
                lds2x64(addr + 48, rr, gg);
                const f32x2 bb = lds64(addr + 64);
                // an invalid pixel takes part with alpha = 0: 1 - alpha = 1, rcp.approx(1) = 1 exactly, so its T, S and both
                // outputs come out unchanged / zero without any further select
                const f32x2 am = pk2(valid0 ? al0 : 0.0f, valid1 ? al1 : 0.0f);
                float om0, om1;
                unpk2(fma2(am, neg2, one2), om0, om1);
                const f32x2 Tf = mul2(pk2(T0, T1), pk2(rcp_approx(om0), rcp_approx(om1)));   // transmittance in front of this record
                const f32x2 d0 = fma2(S0, neg2, rr), d1 = fma2(S1, neg2, gg), d2 = fma2(S2, neg2, bb);
                const f32x2 dLda = mul2(Tf, fma2(d2, G2, fma2(d1, G1, mul2(d0, G0))));
                S0 = fma2(am, d0, S0);
                S1 = fma2(am, d1, S1);
                S2 = fma2(am, d2, S2);
                unpk2(Tf, T0, T1);
                // no gradient through the alpha_max clamp
                float gp0, gp1;
                unpk2(mul2(am, dLda), gp0, gp1);
                gp0 = (raw0 > alpha_max) ? 0.0f : gp0;
                gp1 = (raw1 > alpha_max) ? 0.0f : gp1;
                sts64(taddr, pk2(gp0, gp1));
                sts64(taddr + kGroup * kTStride * 4, mul2(am, Tf));
                taddr += kTStride * 4;
                myq = (k == (lane >> 2)) ? ch * 32 + bit : myq;
                written |= 1u << bit;
                if (++k == kGroup) {
                    reduce_group(sm, warp, lane, kGroup, myq, ox, pya);
                    k = 0;
                    taddr = tbase;
                }
            }
            if (lane == 0) sm.vis[warp][ch] = written;
        }
        if (k) reduce_group(sm, warp, lane, k, myq, ox, pya);
        __syncthreads();
        if (tid < cnt) {
            float m[9];
#pragma unroll
            for (int c = 0; c < 9; ++c) m[c] = 0.f;
            bool any = false;
#pragma unroll
            for (int w = 0; w < kWarps; ++w)
                if ((sm.vis[w][tid >> 5] >> (tid & 31)) & 1u) {
                    any = true;
#pragma unroll
                    for (int c = 0; c < 9; ++c) m[c] += sm.slot[w][tid][c];
                }
            if (any) {
                const Rec& rc = sm.rec[tid];
                const int64_t g = __float_as_int(rc.e.z);
                const float Aq = rc.b.x, Bq = rc.b.z, Cq = rc.c.x;
                // moments about the tile centre -> sums of gp*{dx, dy, dx^2, dx dy, dy^2}, dx = u - x
                const float ut = rc.a.x - xc, vt = rc.a.z - yc;
                const float Dx = fmaf(ut, m[0], -m[1]), Dy = fmaf(vt, m[0], -m[2]);
                const float Dxx = fmaf(ut, Dx - m[1], m[3]);
                const float Dxy = fmaf(vt, Dx, fmaf(-ut, m[2], m[4]));
                const float Dyy = fmaf(vt, Dy - m[2], m[5]);
                const float gu = fmaf(2.0f * Aq, Dx, Bq * Dy) * kLn2;
                const float gv = fmaf(2.0f * Cq, Dy, Bq * Dx) * kLn2;
                if (gu != 0.f) atomicAdd(io.g_means2d + 2 * g, gu);
                if (gv != 0.f) atomicAdd(io.g_means2d + 2 * g + 1, gv);
                if (Dxx != 0.f) atomicAdd(io.g_conics + 3 * g, -0.5f * Dxx);
                if (Dxy != 0.f) atomicAdd(io.g_conics + 3 * g + 1, -Dxy);
                if (Dyy != 0.f) atomicAdd(io.g_conics + 3 * g + 2, -0.5f * Dyy);
                if (m[0] != 0.f) atomicAdd(io.g_opacities + g, m[0] / rc.e.w);
                if (m[6] != 0.f) atomicAdd(io.g_rgbs + 3 * g, m[6]);
                if (m[7] != 0.f) atomicAdd(io.g_rgbs + 3 * g + 1, m[7]);
                if (m[8] != 0.f) atomicAdd(io.g_rgbs + 3 * g + 2, m[8]);
            }
        }
    }
}

// zero the gradient rows of visible entries only (dense zero-fill when radii == nullptr is a memset);
// four entries per thread and load (one 16-byte load when `vec`), two loads in flight per thread
__device__ __forceinline__ void zero_row(int64_t e, float* g_means2d, float* g_conics, float* g_opacities, float* g_rgbs) {
    reinterpret_cast<float2*>(g_means2d)[e] = make_float2(0.f, 0.f);
    g_conics[3 * e] = 0.f; g_conics[3 * e + 1] = 0.f; g_conics[3 * e + 2] = 0.f;
    g_opacities[e] = 0.f;
    g_rgbs[3 * e] = 0.f; g_rgbs[3 * e + 1] = 0.f; g_rgbs[3 * e + 2] = 0.f;
}
__global__ void __launch_bounds__(256) zero_visible_rows_kernel(int64_t n, const int32_t* __restrict__ radii, int vec, float* g_means2d,
                                                                float* g_conics, float* g_opacities, float* g_rgbs) {
    pdl_enter();
    const int64_t q0 = ((int64_t)blockIdx.x * 512 + threadIdx.x) * 4;
    int4 r[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int64_t e = q0 + h * 1024;
        if (vec && e + 4 <= n) {
            r[h] = __ldg(reinterpret_cast<const int4*>(radii + e));
        } else {
            r[h].x = (e < n) ? __ldg(radii + e) : 0;
            r[h].y = (e + 1 < n) ? __ldg(radii + e + 1) : 0;
            r[h].z = (e + 2 < n) ? __ldg(radii + e + 2) : 0;
            r[h].w = (e + 3 < n) ? __ldg(radii + e + 3) : 0;
        }
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int64_t e = q0 + h * 1024;
        if (r[h].x > 0) zero_row(e, g_means2d, g_conics, g_opacities, g_rgbs);
        if (r[h].y > 0) zero_row(e + 1, g_means2d, g_conics, g_opacities, g_rgbs);
        if (r[h].z > 0) zero_row(e + 2, g_means2d, g_conics, g_opacities, g_rgbs);
        if (r[h].w > 0) zero_row(e + 3, g_means2d, g_conics, g_opacities, g_rgbs);
    }
}

// the same from the visibility mask [C][wn] of gs_project_fwd: a lane loads four mask words (16 bytes), the warp then walks
// the non-zero words with lane = bit, so that the rows zeroed together are neighbours in memory
__global__ void __launch_bounds__(256) zero_masked_rows_kernel(int64_t N, int64_t wn, int64_t n_words, const uint32_t* __restrict__ vmask,
                                                               float* g_means2d, float* g_conics, float* g_opacities, float* g_rgbs) {
    pdl_enter();
    const int lane = threadIdx.x & 31;
    const int64_t wi = ((int64_t)blockIdx.x * 256 + threadIdx.x) * 4;              // n_words = C * wn is a multiple of 16
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (wi < n_words) v = __ldg(reinterpret_cast<const uint4*>(vmask + wi));
    if (!__any_sync(0xffffffffu, (v.x | v.y | v.z | v.w) != 0u)) return;
    const int64_t view = wi < n_words ? wi / wn : 0;                               // (a lane's four words belong to one view)
    const int64_t e_lane = view * N + ((wi - view * wn) << 5);                     // entry of bit 0 of this lane's first word
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        uint32_t nz = __ballot_sync(0xffffffffu, w[q] != 0u);
        while (nz) {
            const int s = __ffs(nz) - 1;
            nz &= nz - 1;
            const uint32_t wd = __shfl_sync(0xffffffffu, w[q], s);
            const unsigned int e_lo = __shfl_sync(0xffffffffu, (unsigned int)e_lane, s);   // C * N < 2^31
            if ((wd >> lane) & 1u) zero_row((int64_t)e_lo + 32 * q + lane, g_means2d, g_conics, g_opacities, g_rgbs);
        }
    }
}

__global__ void __launch_bounds__(256) l1_loss_kernel(int64_t n, const float* __restrict__ image, const float* __restrict__ target,
                                                      float* __restrict__ dL, float* loss_sum, float inv_n) {
    pdl_enter();
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


// Measurement aid (bench.py's roofline, outside any timed region): replays the per-pixel decisions of O-R1, one thread per
// pixel, and counts the (pixel, record) pairs the METHOD evaluates -- stats[0] pairs composited; stats[1] pairs the forward
// definition evaluates without compositing (a rule rejects them, or they terminate the pixel); stats[2] pairs the backward
// definition walks (list position <= n_contrib) without compositing; stats[3] records of all tile lists times 256 (the
// dense upper bound).
__global__ void __launch_bounds__(256) pair_stats_kernel(const RasterArgs a, unsigned long long* __restrict__ stats) {
    pdl_enter();
    __shared__ float s_u[256], s_v[256], s_A[256], s_B[256], s_C[256], s_lo[256];
    __shared__ unsigned long long s_sum[3];
    const int tid = threadIdx.x;
    const int64_t bt = blockIdx.x;
    const int64_t view = bt / a.tiles;
    const int t = (int)(bt - view * a.tiles);
    const int ty = t / a.gx, tx = t - ty * a.gx;
    const int j = tx * kTile + (tid & 15), i = ty * kTile + (tid >> 4);
    const bool inside = (i < a.height) && (j < a.width);
    const float px = (float)j + 0.5f, py = (float)i + 0.5f;
    const int64_t start = __ldg(a.ranges + 2 * bt), end = __ldg(a.ranges + 2 * bt + 1);
    if (tid < 3) s_sum[tid] = 0ull;
    float T = 1.0f;
    bool done = !inside;
    unsigned int n_comp = 0, n_rej = 0, n_rej_before_last = 0, rej_run = 0;
    for (int64_t base = start; base < end; base += 256) {
        __syncthreads();
        const int64_t k = base + tid;
        if (k < end) {
            const int g = __ldg(a.vals + k);
            const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + g);
            s_u[tid] = uv.x; s_v[tid] = uv.y;
            s_A[tid] = -0.5f * kLog2e * __ldg(a.conics + 3 * (int64_t)g);
            s_B[tid] = -kLog2e * __ldg(a.conics + 3 * (int64_t)g + 1);
            s_C[tid] = -0.5f * kLog2e * __ldg(a.conics + 3 * (int64_t)g + 2);
            s_lo[tid] = __log2f(__ldg(a.opacities + g));
        }
        __syncthreads();
        const int cnt = (int)((end - base) < 256 ? (end - base) : 256);
        for (int q = 0; q < cnt && !done; ++q) {
            const float e = quad_form(s_A[q], s_B[q], s_C[q], s_u[q] - px, s_v[q] - py);
            const float al = fminf(a.alpha_max, ex2_approx(e + s_lo[q]));
            if (e > 0.0f || al < a.alpha_min) { ++n_rej; ++rej_run; continue; }
            const float Tn = T * (1.0f - al);
            if (Tn < a.t_min) { ++n_rej; done = true; break; }
            T = Tn;
            ++n_comp;
            n_rej_before_last += rej_run;     // rejected pairs in front of the last composited one = what the backward pass walks
            rej_run = 0;
        }
    }
    __syncthreads();
    atomicAdd(&s_sum[0], (unsigned long long)n_comp);
    atomicAdd(&s_sum[1], (unsigned long long)n_rej);
    atomicAdd(&s_sum[2], (unsigned long long)n_rej_before_last);
    __syncthreads();
    if (tid < 3 && s_sum[tid]) atomicAdd(stats + tid, s_sum[tid]);
    if (tid == 3 && end > start) atomicAdd(stats + 3, (unsigned long long)(end - start) * 256ull);
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
    a.filter_thr = cfg->alpha_min > 0.0f ? log2f(cfg->alpha_min) - kFilterMargin : -3.0e38f;
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
    launch_chained(raster_fwd_kernel, dim3((unsigned)(C * a.tiles)), dim3(kBlock), (size_t)(0), (cudaStream_t)stream, a, o);
    return launch_status();
}

extern "C" int gs_raster_bwd(const gs_config* cfg, int32_t C, const gs_camera* cams, int64_t N_total,
                             const int32_t* isect_vals, const int64_t* tile_ranges, const float* means2d, const float* conics,
                             const float* opacities, const float* rgbs, const float* bg, const float* final_T,
                             const int32_t* n_contrib, const float* dL_dimage, const int32_t* radii, const uint32_t* vis_mask,
                             float* dL_dmeans2d, float* dL_dconics, float* dL_dopacities, float* dL_drgbs, void* stream) {
    RasterArgs a;
    int rc = fill_args(cfg, C, cams, isect_vals, tile_ranges, means2d, conics, opacities, rgbs, bg, a);
    if (rc) return rc;
    if (N_total < 0 || N_total >= (1LL << 31)) return GS_ERR_INVALID_ARGUMENT;
    if (!final_T || !n_contrib || !dL_dimage || !dL_dmeans2d || !dL_dconics || !dL_dopacities || !dL_drgbs || !aligned(dL_dmeans2d, 8))
        return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t st = (cudaStream_t)stream;
    if (N_total > 0) {
        if (vis_mask) {
            if (N_total % C != 0 || !aligned(vis_mask, 16)) return GS_ERR_INVALID_ARGUMENT;
            const int64_t N = N_total / C, wn = GS_VIS_WORDS(N), n_words = (int64_t)C * wn;
            launch_chained(zero_masked_rows_kernel, dim3((unsigned)((n_words / 4 + 255) / 256)), dim3(256), (size_t)(0), st, N, wn, n_words, vis_mask, dL_dmeans2d, dL_dconics,
                                                                                          dL_dopacities, dL_drgbs);
            rc = launch_status();
            if (rc) return rc;
        } else if (radii) {
            launch_chained(zero_visible_rows_kernel, dim3((unsigned)((N_total + 2047) / 2048)), dim3(256), (size_t)(0), st, N_total, radii, aligned(radii, 16) ? 1 : 0,
                                                                                           dL_dmeans2d, dL_dconics, dL_dopacities, dL_drgbs);
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
    rc = ensure_smem(raster_bwd_kernel, 0, (int)sizeof(BwdSmem));
    if (rc) return rc;
    launch_chained(raster_bwd_kernel, dim3((unsigned)(C * a.tiles)), dim3(kBlock), (size_t)(sizeof(BwdSmem)), st, a, io);
    return launch_status();
}

extern "C" int gs_raster_pair_stats(const gs_config* cfg, int32_t C, const gs_camera* cams, const int32_t* isect_vals,
                                    const int64_t* tile_ranges, const float* means2d, const float* conics, const float* opacities,
                                    uint64_t* stats, void* stream) {
    RasterArgs a;
    const float bg[3] = {0.f, 0.f, 0.f};
    int rc = fill_args(cfg, C, cams, isect_vals, tile_ranges, means2d, conics, opacities, opacities /*unused*/, bg, a);
    if (rc) return rc;
    if (!stats || !aligned(stats, 8)) return GS_ERR_INVALID_ARGUMENT;
    if (cudaMemsetAsync(stats, 0, 4 * sizeof(uint64_t), (cudaStream_t)stream) != cudaSuccess) return GS_ERR_CUDA;
    launch_chained(pair_stats_kernel, dim3((unsigned)(C * a.tiles)), dim3(256), (size_t)(0), (cudaStream_t)stream, a, reinterpret_cast<unsigned long long*>(stats));
    return launch_status();
}

extern "C" int gs_l1_loss(int64_t n, const float* image, const float* target, float* dL_dimage, float* loss_sum, void* stream) {
    if (n < 0) return GS_ERR_INVALID_ARGUMENT;
    if (n == 0) return GS_OK;
    if (!image || !target || !dL_dimage || !loss_sum) return GS_ERR_INVALID_ARGUMENT;
    const int sms = sm_count();
    int64_t blocks = (n + 255) / 256;
    if (blocks > (int64_t)sms * 16) blocks = (int64_t)sms * 16;
    launch_chained(l1_loss_kernel, dim3((unsigned)blocks), dim3(256), (size_t)(0), (cudaStream_t)stream, n, image, target, dL_dimage, loss_sum, 1.0f / (float)n);
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
