// raster.cu -- per-pixel stages R1 (gs_raster_fwd) and R2 (gs_raster_bwd) plus the harness L1 loss.
//
// One 256-thread block per (view, tile); each of its 8 warps owns an 8x4 pixel block of the 16x16
// tile (lane = pixel).  The tile's sorted records are staged through shared memory in batches of 256
// (one gathered record per thread, conic pre-scaled to the log2 domain).  Only ~1/4 of the (pixel,
// record) pairs of a tile list pass the alpha >= alpha_min rule, so before evaluating anything a
// warp FILTERS the batch: lane l bounds record (chunk*32 + l) over the warp's 8x4 pixel rectangle
// (exact maximum of the concave exponent over the rectangle, conservative margin) and a ballot
// gives the records that can contribute; the warp then walks only those bits.  The filter never
// changes a per-pixel decision, it only skips records for which every pixel would be skipped.
// Forward: a warp stops when all its pixels are saturated, the block stops fetching when every warp
// has.  Backward: back to front from the tile's largest n_contrib; the 9
// partial sums of a record are reduced inside the warp with a value-splitting butterfly (14
// shuffles), written to the warp's own shared-memory slot (shared-memory float atomics are CAS loops
// on this hardware), summed across the 8 warps at the end of the batch and flushed with one
// device-scope red.add per value and (tile, record).
#include "common.cuh"

namespace gs {

constexpr int kBlock = kTile * kTile;  // 256
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

// Can the record contribute to any pixel centre of the rectangle [X0, X0+7] x [Y0, Y0+3]?
// g0 = (u, v, A', B'), g1.x = C', g1.y = log2(opacity).  Exact maximum of the concave exponent over
// the rectangle (inside -> 0, otherwise on the edge(s) facing the mean), compared with a margin.
// The stationary point along an edge uses an approximate reciprocal: an error eps in its position
// lowers the bound by |C'| eps^2, far inside the margin; a NaN (0/0) falls back to the end points.
__device__ __forceinline__ bool rect_may_contribute(const float4 g0, const float4 g1, float X0, float Y0, float thr) {
    const float A = g0.z, B = g0.w, C = g1.x;
    const float dx0 = g0.x - (X0 + 7.0f), dx1 = g0.x - X0;
    const float dy0 = g0.y - (Y0 + 3.0f), dy1 = g0.y - Y0;
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
    return !concave || !(emax + g1.y < thr);
}

// One staged record: 48 bytes of shared memory, conic in the log2 domain.
struct __align__(16) Rec {
    float4 a;   // u, v, A', B'
    float4 b;   // C', log2(opacity), r, g
    float4 c;   // b, opacity, bit pattern of the entry id, unused
};

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
__device__ __forceinline__ float lds32(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}

// gather one record and stage it in the log2 domain
__device__ __forceinline__ void stage_record(const RasterArgs& a, int g, Rec& r) {
    const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + g);
    const float A = __ldg(a.conics + 3 * (int64_t)g), B = __ldg(a.conics + 3 * (int64_t)g + 1), Cc = __ldg(a.conics + 3 * (int64_t)g + 2);
    const float op = __ldg(a.opacities + g);
    r.a = make_float4(uv.x, uv.y, -0.5f * kLog2e * A, -kLog2e * B);
    r.b = make_float4(-0.5f * kLog2e * Cc, __log2f(op), __ldg(a.rgbs + 3 * (int64_t)g), __ldg(a.rgbs + 3 * (int64_t)g + 1));
    r.c = make_float4(__ldg(a.rgbs + 3 * (int64_t)g + 2), op, __int_as_float(g), 0.0f);
}

__global__ void __launch_bounds__(kBlock) raster_fwd_kernel(const RasterArgs a, const RasterFwdOut o) {
    __shared__ Rec s_rec[kBlock];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t bt = blockIdx.x;                  // view * tiles + tile
    const int64_t view = bt / a.tiles;
    const int t = (int)(bt - view * a.tiles);
    const int ty = t / a.gx, tx = t - ty * a.gx;
    const int bx0 = tx * kTile + (warp & 1) * 8, by0 = ty * kTile + (warp >> 1) * 4;   // the warp's 8x4 pixel block
    const int j = bx0 + (lane & 7), i = by0 + (lane >> 3);
    const bool inside = (i < a.height) && (j < a.width);
    const float px = (float)j + 0.5f, py = (float)i + 0.5f;
    const float X0 = (float)bx0 + 0.5f, Y0 = (float)by0 + 0.5f;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(s_rec);
    const float alpha_min = a.alpha_min, alpha_max = a.alpha_max, t_min = a.t_min;

    const int64_t start = __ldg(a.ranges + 2 * bt), end = __ldg(a.ranges + 2 * bt + 1);
    float T = 1.0f, c0 = 0.f, c1 = 0.f, c2 = 0.f;
    int last = 0;
    bool done = !inside;
    for (int64_t base = start; base < end; base += kBlock) {
        if (__syncthreads_and(done)) break;
        const int64_t k = base + tid;
        if (k < end) stage_record(a, __ldg(a.vals + k), s_rec[tid]);
        __syncthreads();
        const int cnt = (int)((end - base) < kBlock ? (end - base) : kBlock);
        const int nbase = (int)(base - start) + 1;
        bool warp_done = __all_sync(0xffffffffu, done);
        for (int ch = 0; ch * 32 < cnt && !warp_done; ++ch) {
            const int r = ch * 32 + lane;
            unsigned int mask = __ballot_sync(0xffffffffu, r < cnt && rect_may_contribute(s_rec[r].a, s_rec[r].b, X0, Y0, a.filter_thr));
            while (mask) {
                const int q = ch * 32 + __ffs(mask) - 1;
                mask &= mask - 1;
                const uint32_t addr = sbase + (uint32_t)q * (uint32_t)sizeof(Rec);
                const float4 ga = lds128(addr);
                const float4 gb = lds128(addr + 16);
                const float bl = lds32(addr + 32);
                const float dx = ga.x - px, dy = ga.y - py;
                const float e = quad_form(ga.z, ga.w, gb.x, dx, dy);
                const float alpha = fminf(alpha_max, ex2_approx(e + gb.y));
                const float Tn = T * (1.0f - alpha);
                const bool ok = !done && !(e > 0.0f) && !(alpha < alpha_min);
                const bool term = ok && (Tn < t_min);
                const bool upd = ok && !term;
                const float wgt = upd ? alpha * T : 0.0f;
                c0 = fmaf(gb.z, wgt, c0);
                c1 = fmaf(gb.w, wgt, c1);
                c2 = fmaf(bl, wgt, c2);
                T = upd ? Tn : T;
                last = upd ? nbase + q : last;
                done = done || term;
                if (__all_sync(0xffffffffu, done)) { warp_done = true; break; }
            }
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

// ---- backward reduction ----------------------------------------------------------------------
// Per (pixel, record) pair the backward pass produces two scalars: gp = dL/dpower and wgt = alpha*T
// (the weight of dL/dimage in dL/drgb).  Every per-record sum is a contraction of those over the
// pixels: with pixel offsets (x, y) from the tile centre, the geometric gradients need the moments
// sum gp*{1, x, y, x^2, xy, y^2} and dL/drgb needs sum wgt*g_c -- 9 values.  Instead of a 32-lane
// butterfly per record (14 shuffles), a warp TRANSPOSES: lane = pixel writes (gp, wgt) of up to 8
// records into a shared-memory tile, then lane (record g, pixel row t) reads its row of 8 pixels
// (2+2 LDS.128), accumulates the moments with immediate x offsets (FFMA), and only the 4 lanes of a
// record are combined by shuffles (value-splitting, 8 shuffles per 8 records).
#ifndef GS_BWD_BATCH
#define GS_BWD_BATCH 64
#endif
constexpr int kBwdBatch = GS_BWD_BATCH;     // records staged per batch in the backward kernel
constexpr int kBwdChunks = kBwdBatch / 32;
constexpr int kWarps = kBlock / 32;
constexpr int kGroup = 8;                   // records reduced together by one warp
constexpr int kTStride = 36;                // floats per transposition row: 32 pixels + 4 (bank spread for LDS.128)
constexpr int kGStride = 28;                // floats per row of staged dL/dimage: 3 x 8 + 4
constexpr int kSlot = 9;                    // floats per (warp, record) slot (odd stride: conflict-free flush)

struct BwdSmem {
    Rec rec[kBwdBatch];
    float slot[kWarps][kBwdBatch][kSlot];   // m0, m1x, m1y, m2xx, m2xy, m2yy, dr, dg, (db at [8])
    float tbuf[kWarps][2 * kGroup][kTStride];   // rows 0..7: gp of record k over the warp's 32 pixels; rows 8..15: wgt
    float gpix[kWarps][4][kGStride];        // dL/dimage of the warp's pixels: row t holds g0[8], g1[8], g2[8]
    unsigned int vis[kWarps][kBwdChunks];   // which records of the batch a warp wrote
    int max_contrib;
};

__device__ __forceinline__ void sts32(uint32_t addr, float v) {
    asm volatile("st.shared.f32 [%0], %1;" :: "r"(addr), "f"(v));
}

// Reduce the k (<= 8) records of a warp's group; `pyt` = this lane's row offset from the tile centre
// (lane = 4*g + t: record g, pixel row t), `ox` = x offset of the warp's 8 columns' centre.
// `myq` = position in the batch of record g.
__device__ __forceinline__ void reduce_group(BwdSmem& sm, int warp, int lane, int k, int myq, float ox, float pyt) {
    __syncwarp();
    const int g = lane >> 2, t = lane & 3;
    const uint32_t tb = (uint32_t)__cvta_generic_to_shared(&sm.tbuf[warp][g][t * 8]);
    const float4 p0 = lds128(tb), p1 = lds128(tb + 16);
    const float4 w0 = lds128(tb + kGroup * kTStride * 4), w1 = lds128(tb + kGroup * kTStride * 4 + 16);
    const uint32_t gb = (uint32_t)__cvta_generic_to_shared(&sm.gpix[warp][t][0]);
    // moments of gp over the row, x measured from the centre of the 8 columns (-3.5 .. 3.5)
    const float a0 = p0.x + p1.w, a1 = p0.y + p1.z, a2 = p0.z + p1.y, a3 = p0.w + p1.x;
    const float d0 = p1.w - p0.x, d1 = p1.z - p0.y, d2 = p1.y - p0.z, d3 = p1.x - p0.w;
    const float s0 = (a0 + a1) + (a2 + a3);
    const float s1 = fmaf(3.5f, d0, fmaf(2.5f, d1, fmaf(1.5f, d2, 0.5f * d3)));
    const float s2 = fmaf(12.25f, a0, fmaf(6.25f, a1, fmaf(2.25f, a2, 0.25f * a3)));
    float v[9];
    // shift to the tile centre: x_t = x + ox, y_t = pyt
    const float m1x = fmaf(ox, s0, s1);
    v[0] = s0;
    v[1] = m1x;
    v[2] = pyt * s0;
    v[3] = fmaf(ox, m1x + s1, s2);          // s2 + 2 ox s1 + ox^2 s0
    v[4] = pyt * m1x;
    v[5] = pyt * v[2];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float4 ga = lds128(gb + c * 32), gc = lds128(gb + c * 32 + 16);
        float acc = w0.x * ga.x;
        acc = fmaf(w0.y, ga.y, acc); acc = fmaf(w0.z, ga.z, acc); acc = fmaf(w0.w, ga.w, acc);
        acc = fmaf(w1.x, gc.x, acc); acc = fmaf(w1.y, gc.y, acc); acc = fmaf(w1.z, gc.z, acc); acc = fmaf(w1.w, gc.w, acc);
        v[6 + c] = acc;
    }
    // combine the 4 rows (lanes t = 0..3 of the record): values 0..7 split, value 8 plain
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
    // lane t now holds values (4*b1 + 2*b0, +1) = (2*tt, 2*tt + 1) with tt = 2*b1 + b0 = t
    if (g < k) {
        float* slot = &sm.slot[warp][myq][0];
        slot[2 * t] = e0;
        slot[2 * t + 1] = e1;
        if (t == 0) slot[8] = w;
    }
    __syncwarp();
}

__global__ void __launch_bounds__(kBlock) raster_bwd_kernel(const RasterArgs a, const RasterBwdIO io) {
    extern __shared__ __align__(16) unsigned char bwd_smem_raw[];
    BwdSmem& sm = *reinterpret_cast<BwdSmem*>(bwd_smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t bt = blockIdx.x;
    const int64_t view = bt / a.tiles;
    const int t = (int)(bt - view * a.tiles);
    const int ty = t / a.gx, tx = t - ty * a.gx;
    const int bx0 = tx * kTile + (warp & 1) * 8, by0 = ty * kTile + (warp >> 1) * 4;
    const int j = bx0 + (lane & 7), i = by0 + (lane >> 3);
    const bool inside = (i < a.height) && (j < a.width);
    const float px = (float)j + 0.5f, py = (float)i + 0.5f;
    const float X0 = (float)bx0 + 0.5f, Y0 = (float)by0 + 0.5f;
    const float xc = (float)(tx * kTile + kTile / 2), yc = (float)(ty * kTile + kTile / 2);   // tile centre
    const float ox = (warp & 1) ? 4.0f : -4.0f;                                            // centre of the warp's columns - xc
    const float pyt = (float)((warp >> 1) * 4 + (lane & 3)) + 0.5f - 8.0f;                 // reduce-phase row (lane & 3) - yc
    const int64_t start = __ldg(a.ranges + 2 * bt);
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(sm.rec);
    const uint32_t tbase = (uint32_t)__cvta_generic_to_shared(&sm.tbuf[warp][0][lane]);
    const float alpha_min = a.alpha_min, alpha_max = a.alpha_max;

    float T = 0.f, g0 = 0.f, g1 = 0.f, g2 = 0.f;
    int ncon = 0;
    if (inside) {
        const int64_t pix = (view * a.height + i) * a.width + j;
        T = __ldg(io.final_T + pix);
        ncon = __ldg(io.n_contrib + pix);
        g0 = __ldg(io.dL_dimage + 3 * pix); g1 = __ldg(io.dL_dimage + 3 * pix + 1); g2 = __ldg(io.dL_dimage + 3 * pix + 2);
    }
    {
        float* gr = &sm.gpix[warp][lane >> 3][lane & 7];
        gr[0] = g0; gr[8] = g1; gr[16] = g2;
    }
    if (tid == 0) sm.max_contrib = 0;
    __syncthreads();
    int wmax = ncon;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, d));
    if (lane == 0 && wmax > 0) atomicMax(&sm.max_contrib, wmax);
    __syncthreads();
    const int maxn = sm.max_contrib;
    if (maxn == 0) return;
    // colour accumulated behind the current record
    float S0 = a.bg0, S1 = a.bg1, S2 = a.bg2;
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
            const int cbase = b * kBwdBatch + ch * 32;          // list position of bit 0 of this chunk
            unsigned int mask = __ballot_sync(0xffffffffu, r < cnt && (cbase + lane) < wmax &&
                                                               rect_may_contribute(sm.rec[r].a, sm.rec[r].b, X0, Y0, a.filter_thr));
            const int nrel = ncon - cbase;                      // this pixel walks bits < nrel
            unsigned int written = 0;
            const uint32_t cbase_addr = sbase + (uint32_t)(ch * 32) * (uint32_t)sizeof(Rec);
            while (mask) {
                const int bit = msb(mask);
                mask ^= 1u << bit;
                const uint32_t addr = cbase_addr + (uint32_t)bit * (uint32_t)sizeof(Rec);
                const float4 ga = lds128(addr);
                const float4 gb = lds128(addr + 16);
                const float dx = ga.x - px, dy = ga.y - py;
                const float e = quad_form(ga.z, ga.w, gb.x, dx, dy);
                const float raw = ex2_approx(e + gb.y);
                const float alpha = fminf(alpha_max, raw);
                const bool valid = (bit < nrel) && !(e > 0.0f) && !(alpha < alpha_min);
                if (!__any_sync(0xffffffffu, valid)) continue;
                const float cb = lds32(addr + 32);
                // quantities of an invalid lane are computed but selected away
                const float Tf = T * rcp_approx(1.0f - alpha);   // transmittance in front of this record
                const float d0 = gb.z - S0, d1 = gb.w - S1, d2 = cb - S2;
                const float dL_dalpha = Tf * fmaf(d2, g2, fmaf(d1, g1, d0 * g0));
                const float am = valid ? alpha : 0.0f;
                S0 = fmaf(am, d0, S0);
                S1 = fmaf(am, d1, S1);
                S2 = fmaf(am, d2, S2);
                T = valid ? Tf : T;
                // no gradient through the alpha_max clamp
                const float gp = (raw > alpha_max) ? 0.0f : am * dL_dalpha;   // dL/dpower
                sts32(taddr, gp);
                sts32(taddr + kGroup * kTStride * 4, am * Tf);
                taddr += kTStride * 4;
                myq = (k == (lane >> 2)) ? ch * 32 + bit : myq;
                written |= 1u << bit;
                if (++k == kGroup) {
                    reduce_group(sm, warp, lane, kGroup, myq, ox, pyt);
                    k = 0;
                    taddr = tbase;
                }
            }
            if (lane == 0) sm.vis[warp][ch] = written;
        }
        if (k) reduce_group(sm, warp, lane, k, myq, ox, pyt);
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
                const int64_t g = __float_as_int(rc.c.z);
                // moments about the tile centre -> sums of gp*{dx, dy, dx^2, dx dy, dy^2}, dx = u - x
                const float ut = rc.a.x - xc, vt = rc.a.y - yc;
                const float Dx = fmaf(ut, m[0], -m[1]), Dy = fmaf(vt, m[0], -m[2]);
                const float Dxx = fmaf(ut, Dx - m[1], m[3]);                       // ut^2 m0 - 2 ut m1x + m2xx
                const float Dxy = fmaf(vt, Dx, fmaf(-ut, m[2], m[4]));             // ut vt m0 - vt m1x - ut m1y + m2xy
                const float Dyy = fmaf(vt, Dy - m[2], m[5]);
                // A dx + B dy = -(2A' dx + B' dy) ln 2 with the staged log2-domain conic
                const float gu = fmaf(2.0f * rc.a.z, Dx, rc.a.w * Dy) * kLn2;
                const float gv = fmaf(2.0f * rc.b.x, Dy, rc.a.w * Dx) * kLn2;
                if (gu != 0.f) atomicAdd(io.g_means2d + 2 * g, gu);
                if (gv != 0.f) atomicAdd(io.g_means2d + 2 * g + 1, gv);
                if (Dxx != 0.f) atomicAdd(io.g_conics + 3 * g, -0.5f * Dxx);
                if (Dxy != 0.f) atomicAdd(io.g_conics + 3 * g + 1, -Dxy);
                if (Dyy != 0.f) atomicAdd(io.g_conics + 3 * g + 2, -0.5f * Dyy);
                if (m[0] != 0.f) atomicAdd(io.g_opacities + g, m[0] / rc.c.y);
                if (m[6] != 0.f) atomicAdd(io.g_rgbs + 3 * g, m[6]);
                if (m[7] != 0.f) atomicAdd(io.g_rgbs + 3 * g + 1, m[7]);
                if (m[8] != 0.f) atomicAdd(io.g_rgbs + 3 * g + 2, m[8]);
            }
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
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(raster_bwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BwdSmem)) != cudaSuccess)
            return GS_ERR_CUDA;
        attr_set = true;
    }
    raster_bwd_kernel<<<(unsigned)(C * a.tiles), kBlock, sizeof(BwdSmem), st>>>(a, io);
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
