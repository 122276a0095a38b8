// binning.cu -- tile binning B1..B4 (gs_bin_tiles) and the stand-alone radix sort (gs_sort_pairs).
//
// The result defined by SURVEY.md 8(c) O-B is the list of (tile | depth, entry) records in stable
// key order.  A stable sort by the 64-bit key (tile << 32 | depth) equals a stable sort by depth
// followed by a stable sort by tile, and only the second one has to touch the M records (M is 19..80
// times the number V of visible entries).  So the work is split in two levels:
//
//   compact_kernel     B1a: visible entries (radius > 0, >= 1 tile) in ascending entry order ->
//                      (view << 32 | depth bits, entry); ordered chained scan (decoupled look-back).
//   hist_kernel +      depth sort of the V compacted entries: stable LSD radix sort on the depth bits
//   onesweep_kernel    and the view bits (64-bit keys, 8-bit digits; also serves gs_sort_pairs).
//   emit_kernel        B1b+B2: per-entry tile counts scanned in DEPTH order (ordered chained scan), one
//                      (32-bit tile id, entry) record per overlapped tile, written warp-cooperatively;
//                      the digit histograms of the tile sort are accumulated on the fly.
//   scan_hist_kernel   exclusive scan of those histograms -> global digit bases.
//   tile_sweep_kernel  B3: stable LSD radix sort of the M records on the tile id only: 2 passes of 8 or
//                      9 bits for every BASELINE configuration (one read + one write of 8 bytes per
//                      record and pass), persistent blocks, per-digit decoupled look-back.
//   ranges_kernel      B4: per-tile [start, end) from the sorted tile ids.
//   keys_kernel        optional: the 64-bit keys (tile << 32 | depth bits) of the sorted records.
//
// Equal (tile, depth) records keep ascending entry order (reading A10) because every step is
// order-preserving: index-ordered compaction, stable depth sort, depth-ordered emit, stable tile sort.
// The counts V and M live in device memory; no stage needs the host.
#include "common.cuh"

namespace gs {

// ------------------------------------------------------------------------------ workspace layout
struct BinHeader {
    unsigned long long M;          // records the batch needs (sum of tile counts of all visible entries)
    unsigned long long V;          // visible entries (clamped to the compact capacity)
    unsigned long long n_rec;      // records actually emitted = min(M, capacity_M)
    unsigned long long M_acc;      // accumulator behind M
    unsigned int compact_done;
    unsigned int emit_ticket;
    unsigned int sort_ticket[8];   // depth-sort passes
    unsigned int tsort_ticket[4];  // tile-sort passes
    unsigned int compact_ticket;
    unsigned int pad;
};
static_assert(sizeof(BinHeader) == 96, "header size");

constexpr int kRadix = 256;            // depth sort: 8-bit digits
constexpr int kMaxPasses = 8;

constexpr int kScanThreads = 256;      // compact / emit: 4 entries per thread
constexpr int kScanItems = 4;
constexpr int kScanTile = kScanThreads * kScanItems;

constexpr int kSortThreads = 256;      // depth sort
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSortItems = 16;
constexpr int kSortTile = kSortThreads * kSortItems;

constexpr int kTsThreads = 512;        // tile sort
constexpr int kTsWarps = kTsThreads / 32;
constexpr int kTsItems = 8;
constexpr int kTsTile = kTsThreads * kTsItems;
constexpr int kTsMaxBits = 9;
constexpr int kTsMaxBins = 1 << kTsMaxBits;
constexpr int kTsMaxPasses = 4;

struct SortPlan {
    int P;
    int shift[kMaxPasses];
    unsigned int mask[kMaxPasses];
};

// tile sort: P passes of `bits` (8 or 9) wide digits starting at bit 0 of the 32-bit tile id
struct TilePlan {
    int P;
    int bits;
    int shift[kTsMaxPasses];
    unsigned int mask[kTsMaxPasses];
};

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Workspace {
    size_t off_header, off_hist, off_thist, off_compact_status, off_emit_status, off_sort_status, off_tsort_status, zero_bytes;
    size_t off_ckeys0, off_ckeys1, off_cvals0, off_cvals1, off_tkeys0, off_tkeys1, off_vals, total;
    int64_t vcap;
};
static Workspace layout(int64_t n_entries, int64_t capacity) {
    Workspace w;
    // every visible entry emits >= 1 record, so V <= M; a call that fits capacity has V <= capacity
    w.vcap = n_entries < capacity ? n_entries : capacity;
    if (w.vcap < 1) w.vcap = 1;
    size_t o = 0;
    w.off_header = o; o += sizeof(BinHeader);
    o = align_up(o, 256);
    w.off_hist = o; o += (size_t)kMaxPasses * kRadix * sizeof(unsigned int);
    w.off_thist = o; o += (size_t)kTsMaxPasses * kTsMaxBins * sizeof(unsigned int);
    o = align_up(o, 256);
    w.off_compact_status = o; o += (size_t)((n_entries + kScanTile - 1) / kScanTile + 1) * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.off_emit_status = o; o += (size_t)((w.vcap + kScanTile - 1) / kScanTile + 1) * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.off_sort_status = o; o += (size_t)((w.vcap + kSortTile - 1) / kSortTile + 1) * kRadix * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.off_tsort_status = o; o += (size_t)((capacity + kTsTile - 1) / kTsTile + 1) * kTsMaxBins * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.zero_bytes = o;  // everything up to here is cleared at the start of a call
    w.off_ckeys0 = o; o += (size_t)w.vcap * sizeof(uint64_t); o = align_up(o, 256);
    w.off_ckeys1 = o; o += (size_t)w.vcap * sizeof(uint64_t); o = align_up(o, 256);
    w.off_cvals0 = o; o += (size_t)w.vcap * sizeof(int32_t); o = align_up(o, 256);
    w.off_cvals1 = o; o += (size_t)w.vcap * sizeof(int32_t); o = align_up(o, 256);
    w.off_tkeys0 = o; o += (size_t)capacity * sizeof(uint32_t); o = align_up(o, 256);
    w.off_tkeys1 = o; o += (size_t)capacity * sizeof(uint32_t); o = align_up(o, 256);
    w.off_vals = o; o += (size_t)capacity * sizeof(int32_t); o = align_up(o, 256);
    w.total = o;
    return w;
}

static SortPlan make_plan(int end_bit, bool skip_bit31) {
    SortPlan p;
    p.P = 0;
    const int low_end = end_bit < 32 ? end_bit : (skip_bit31 ? 31 : 32);
    for (int b = 0; b < low_end; b += 8) {
        const int w = low_end - b < 8 ? low_end - b : 8;
        p.shift[p.P] = b; p.mask[p.P] = (1u << w) - 1u; ++p.P;
    }
    if (end_bit > 32) {
        const int nb = end_bit - 32;
        const int np = (nb + 7) / 8;
        int b = 32;
        for (int k = 0; k < np; ++k) {
            const int w = nb / np + (k < nb % np ? 1 : 0);
            p.shift[p.P] = b; p.mask[p.P] = (1u << w) - 1u; ++p.P;
            b += w;
        }
    }
    return p;
}

static TilePlan make_tile_plan(int tile_bits) {
    TilePlan p;
    const int p8 = (tile_bits + 7) / 8, p9 = (tile_bits + 8) / 9;
    p.bits = p9 < p8 ? 9 : 8;
    p.P = p9 < p8 ? p9 : p8;
    int b = 0;
    for (int k = 0; k < p.P; ++k) {
        const int w = tile_bits / p.P + (k < tile_bits % p.P ? 1 : 0);   // widths differ by at most one bit
        p.shift[k] = b; p.mask[k] = (1u << w) - 1u;
        b += w;
    }
    return p;
}

// ------------------------------------------------------------------------------ device helpers
__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_volatile_u64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long shfl_up_u64(unsigned long long v, int d) {
    unsigned int lo = (unsigned int)v, hi = (unsigned int)(v >> 32);
    lo = __shfl_up_sync(0xffffffffu, lo, d);
    hi = __shfl_up_sync(0xffffffffu, hi, d);
    return ((unsigned long long)hi << 32) | lo;
}
__device__ __forceinline__ unsigned long long shfl_u64(unsigned long long v, int src) {
    unsigned int lo = (unsigned int)v, hi = (unsigned int)(v >> 32);
    lo = __shfl_sync(0xffffffffu, lo, src);
    hi = __shfl_sync(0xffffffffu, hi, src);
    return ((unsigned long long)hi << 32) | lo;
}

constexpr unsigned long long kFlagAgg = 1ull << 62;
constexpr unsigned long long kFlagIncl = 2ull << 62;
constexpr unsigned long long kValMask = (1ull << 62) - 1ull;

// Ordered chained scan step (warp 0 of a block): publish this block's total, look back over the
// preceding blocks (32 at a time) until an inclusive prefix is found, publish the own inclusive
// prefix, return the exclusive one.  `tile` is the block's position in ticket order.
__device__ __forceinline__ unsigned long long chained_scan_lookback(unsigned long long* status, int64_t tile,
                                                                     unsigned long long block_total, int lane) {
    unsigned long long excl = 0;
    if (tile == 0) {
        if (lane == 0) st_volatile_u64(status, kFlagIncl | block_total);
        return 0;
    }
    if (lane == 0) st_volatile_u64(status + tile, kFlagAgg | block_total);
    int64_t look = tile - 1;
    while (true) {
        const int64_t idx = look - lane;
        unsigned long long st = kFlagIncl;   // virtual predecessor of block 0: inclusive 0
        if (idx >= 0) {
            do { st = ld_volatile_u64(status + idx); } while ((st >> 62) == 0);
        }
        const unsigned int incl = __ballot_sync(0xffffffffu, (st >> 62) == 2);
        unsigned long long v = st & kValMask;
        if (incl) {
            const int first = __ffs(incl) - 1;
            if (lane > first) v = 0;
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v += shfl_u64(v, lane ^ d);
        excl += v;
        if (incl) break;
        look -= 32;
    }
    if (lane == 0) st_volatile_u64(status + tile, kFlagIncl | (excl + block_total));
    return excl;
}

// ------------------------------------------------------------------------------ B1a: compaction
struct CompactArgs {
    int64_t n_entries;      // C * N
    int64_t N;
    int32_t gx, gy;
    const float* means2d; const float* depths; const int32_t* radii;
    int64_t vcap;
    unsigned long long* ckeys; int32_t* cvals;
    BinHeader* hdr;
    unsigned long long* status;
    unsigned int n_blocks;
    unsigned long long* M_dev;
};

__global__ void __launch_bounds__(kScanThreads) compact_kernel(const CompactArgs a) {
    __shared__ unsigned int s_ticket;
    __shared__ unsigned long long s_base;
    __shared__ unsigned long long s_warp_tiles[kScanThreads / 32];
    __shared__ unsigned int s_warp_vis[kScanThreads / 32];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_ticket = atomicAdd(&a.hdr->compact_ticket, 1u);
    __syncthreads();
    const int64_t tile = s_ticket;
    const int64_t e0 = tile * kScanTile + (int64_t)tid * kScanItems;

    int rad[kScanItems];
    if (e0 + kScanItems <= a.n_entries) {
        const int4 r4 = __ldg(reinterpret_cast<const int4*>(a.radii + e0));
        rad[0] = r4.x; rad[1] = r4.y; rad[2] = r4.z; rad[3] = r4.w;
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) rad[k] = (e0 + k < a.n_entries) ? __ldg(a.radii + e0 + k) : 0;
    }
    unsigned long long key[kScanItems];
    bool vis[kScanItems];
    unsigned long long t_tiles = 0;
    unsigned int t_vis = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        vis[k] = false; key[k] = 0;
        if (rad[k] > 0) {
            const int64_t e = e0 + k;
            const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + e);
            int x0, x1, y0, y1;
            tile_rect(uv.x, uv.y, rad[k], a.gx, a.gy, x0, x1, y0, y1);
            const unsigned int cnt = (unsigned int)(x1 - x0) * (unsigned int)(y1 - y0);
            if (cnt) {
                const unsigned long long view = (unsigned long long)(e / a.N);
                key[k] = (view << 32) | (unsigned long long)__float_as_uint(__ldg(a.depths + e));
                vis[k] = true;
                t_tiles += cnt;
                ++t_vis;
            }
        }
    }
    // block totals; exclusive scan of the visible count
    unsigned int inc_v = t_vis;
    unsigned long long sum_t = t_tiles;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned int ov = __shfl_up_sync(0xffffffffu, inc_v, d);
        if (lane >= d) inc_v += ov;
        sum_t += shfl_u64(sum_t, lane ^ d);
    }
    if (lane == 31) { s_warp_vis[warp] = inc_v; s_warp_tiles[warp] = sum_t; }
    __syncthreads();
    unsigned int wbase_v = 0, block_vis = 0;
    unsigned long long block_tiles = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) {
        if (w < warp) wbase_v += s_warp_vis[w];
        block_vis += s_warp_vis[w];
        block_tiles += s_warp_tiles[w];
    }
    if (warp == 0) {
        const unsigned long long excl = chained_scan_lookback(a.status, tile, block_vis, lane);
        if (lane == 0) {
            s_base = excl;
            // total record count: unordered sum, published by whichever block finishes last
            atomicAdd(&a.hdr->M_acc, block_tiles);
            __threadfence();
            const unsigned int done = atomicAdd(&a.hdr->compact_done, 1u);
            if (done == a.n_blocks - 1) {
                __threadfence();
                const unsigned long long M = ld_volatile_u64(&a.hdr->M_acc);
                a.hdr->M = M;
                if (a.M_dev) *a.M_dev = M;
            }
            if (tile == (int64_t)a.n_blocks - 1) {
                const unsigned long long V = excl + block_vis;
                a.hdr->V = V < (unsigned long long)a.vcap ? V : (unsigned long long)a.vcap;
            }
        }
    }
    __syncthreads();
    unsigned long long pos = s_base + wbase_v + inc_v - t_vis;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k)
        if (vis[k]) {
            if (pos < (unsigned long long)a.vcap) {
                a.ckeys[pos] = key[k];
                a.cvals[pos] = (int)(e0 + k);
            }
            ++pos;
        }
}

// ------------------------------------------------------------------------------ B1b + B2: emit
struct EmitArgs {
    int64_t N;
    int32_t gx, gy;
    unsigned int tiles;            // gx * gy
    const float* means2d; const int32_t* radii;
    const int32_t* cvals;          // visible entries in (view, depth, entry) order
    int64_t capacity;
    unsigned int* tkeys; int32_t* vals;
    BinHeader* hdr;
    unsigned long long* status;
    unsigned int* thist;           // [P][kTsMaxBins]
    TilePlan plan;
};

constexpr unsigned int kEmitBig = 2048;   // entries with more records than this are written by the whole block

__device__ __forceinline__ void emit_record(const EmitArgs& a, unsigned int* s_hist, unsigned long long pos, unsigned int k,
                                            unsigned int w, float inv_w, unsigned int t0, int id) {
    // k -> (row, column) of the tile rectangle: reciprocal estimate, then an exact fix-up
    unsigned int ry = (unsigned int)(((float)k + 0.5f) * inv_w);
    int rx = (int)(k - ry * w);
    if (rx < 0) { --ry; rx += (int)w; }
    else if (rx >= (int)w) { ++ry; rx -= (int)w; }
    const unsigned int t = t0 + ry * (unsigned int)a.gx + (unsigned int)rx;
    if (pos < (unsigned long long)a.capacity) {   // records beyond the capacity are dropped (and not counted)
#pragma unroll
        for (int p = 0; p < kTsMaxPasses; ++p)
            if (p < a.plan.P) atomicAdd(&s_hist[p * kTsMaxBins + ((t >> a.plan.shift[p]) & a.plan.mask[p])], 1u);
        a.tkeys[pos] = t;
        a.vals[pos] = id;
    }
}

__global__ void __launch_bounds__(kScanThreads) emit_kernel(const EmitArgs a) {
    __shared__ unsigned int s_ticket;
    __shared__ unsigned long long s_base;
    __shared__ unsigned long long s_warp_tiles[kScanThreads / 32];
    __shared__ unsigned long long s_off[kScanTile];   // record offset of the entry within the block
    __shared__ unsigned int s_cnt[kScanTile];
    __shared__ unsigned int s_t0[kScanTile];          // tile id of the rectangle's first tile
    __shared__ unsigned int s_w[kScanTile];
    __shared__ int s_id[kScanTile];
    __shared__ unsigned int s_big[kScanTile];
    __shared__ unsigned int s_nbig;
    __shared__ unsigned int s_hist[kTsMaxPasses * kTsMaxBins];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int k = tid; k < a.plan.P * kTsMaxBins; k += kScanThreads) s_hist[k] = 0;
    const unsigned long long V = a.hdr->V;
    const int64_t n_blocks = (int64_t)((V + kScanTile - 1) / kScanTile);
    while (true) {
        __syncthreads();   // shared arrays of the previous tile are no longer read
        if (tid == 0) { s_ticket = atomicAdd(&a.hdr->emit_ticket, 1u); s_nbig = 0; }
        __syncthreads();
        const int64_t tile = s_ticket;
        if (tile >= n_blocks) break;
        const int64_t j0 = tile * kScanTile + (int64_t)tid * kScanItems;
        int id[kScanItems];
        if (j0 + kScanItems <= (int64_t)V) {
            const int4 v4 = __ldg(reinterpret_cast<const int4*>(a.cvals + j0));
            id[0] = v4.x; id[1] = v4.y; id[2] = v4.z; id[3] = v4.w;
        } else {
#pragma unroll
            for (int k = 0; k < kScanItems; ++k) id[k] = (j0 + k < (int64_t)V) ? __ldg(a.cvals + j0 + k) : -1;
        }
        unsigned int cnt[kScanItems], t0[kScanItems], ww[kScanItems];
        unsigned long long t_tiles = 0;
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) {
            cnt[k] = 0; t0[k] = 0; ww[k] = 1;
            if (id[k] >= 0) {
                const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + id[k]);
                const int rad = __ldg(a.radii + id[k]);
                int x0, x1, y0, y1;
                tile_rect(uv.x, uv.y, rad, a.gx, a.gy, x0, x1, y0, y1);
                ww[k] = (unsigned int)(x1 - x0);
                cnt[k] = ww[k] * (unsigned int)(y1 - y0);
                const unsigned int view = (unsigned int)((int64_t)id[k] / a.N);
                t0[k] = view * a.tiles + (unsigned int)y0 * (unsigned int)a.gx + (unsigned int)x0;
                t_tiles += cnt[k];
            }
        }
        unsigned long long inc_t = t_tiles;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned long long ot = shfl_up_u64(inc_t, d);
            if (lane >= d) inc_t += ot;
        }
        if (lane == 31) s_warp_tiles[warp] = inc_t;
        __syncthreads();
        unsigned long long wbase_t = 0, block_tiles = 0;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) {
            if (w < warp) wbase_t += s_warp_tiles[w];
            block_tiles += s_warp_tiles[w];
        }
        unsigned long long off = wbase_t + inc_t - t_tiles;   // exclusive
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) {
            const int ci = tid * kScanItems + k;
            s_off[ci] = off; s_cnt[ci] = cnt[k]; s_t0[ci] = t0[k]; s_w[ci] = ww[k]; s_id[ci] = id[k];
            if (cnt[k] > kEmitBig) s_big[atomicAdd(&s_nbig, 1u)] = (unsigned int)ci;
            off += cnt[k];
        }
        if (warp == 0) {
            const unsigned long long excl = chained_scan_lookback(a.status, tile, block_tiles, lane);
            if (lane == 0) {
                s_base = excl;
                if (tile == n_blocks - 1) {
                    const unsigned long long tot = excl + block_tiles;
                    a.hdr->n_rec = tot < (unsigned long long)a.capacity ? tot : (unsigned long long)a.capacity;
                }
            }
        }
        __syncthreads();
        const unsigned long long base = s_base;
        const int64_t rem = (int64_t)V - tile * kScanTile;
        const int nvalid = (int)(rem < kScanTile ? rem : kScanTile);
        // warp-cooperative emit: each warp takes entries round-robin, its 32 lanes write the entry's
        // records to consecutive addresses
        for (int j = warp; j < nvalid; j += kScanThreads / 32) {
            const unsigned int c = s_cnt[j];
            if (c > kEmitBig) continue;
            const unsigned int w = s_w[j], tt0 = s_t0[j];
            const unsigned long long o = base + s_off[j];
            const int e = s_id[j];
            const float inv_w = 1.0f / (float)w;
            for (unsigned int k = lane; k < c; k += 32) emit_record(a, s_hist, o + k, k, w, inv_w, tt0, e);
        }
        // very large entries (whole-screen splats): the whole block writes them
        const unsigned int nbig = s_nbig;
        for (unsigned int b = 0; b < nbig; ++b) {
            const int j = (int)s_big[b];
            const unsigned int c = s_cnt[j], w = s_w[j], tt0 = s_t0[j];
            const unsigned long long o = base + s_off[j];
            const int e = s_id[j];
            const float inv_w = 1.0f / (float)w;
            for (unsigned int k = tid; k < c; k += kScanThreads) emit_record(a, s_hist, o + k, k, w, inv_w, tt0, e);
        }
    }
    __syncthreads();
    for (int k = tid; k < a.plan.P * kTsMaxBins; k += kScanThreads) {
        const unsigned int v = s_hist[k];
        if (v) atomicAdd(a.thist + k, v);
    }
}

// exclusive scan of the tile-sort digit histograms (one block; P * kTsMaxBins values)
__global__ void __launch_bounds__(kTsMaxBins) scan_hist_kernel(unsigned int* thist, int P) {
    __shared__ unsigned int s[kTsMaxBins];
    const int tid = threadIdx.x;
    for (int p = 0; p < P; ++p) {
        const unsigned int v = thist[p * kTsMaxBins + tid];
        s[tid] = v;
        __syncthreads();
        for (int d = 1; d < kTsMaxBins; d <<= 1) {
            const unsigned int o = tid >= d ? s[tid - d] : 0u;
            __syncthreads();
            s[tid] += o;
            __syncthreads();
        }
        thist[p * kTsMaxBins + tid] = s[tid] - v;
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------ histograms
__global__ void __launch_bounds__(256) hist_kernel(const uint64_t* __restrict__ keys, const unsigned long long* count, int64_t capacity,
                                                   const SortPlan plan, unsigned int* __restrict__ hist) {
    __shared__ unsigned int h[kMaxPasses][kRadix];
    for (int k = threadIdx.x; k < kMaxPasses * kRadix; k += blockDim.x) (&h[0][0])[k] = 0;
    __syncthreads();
    const unsigned long long M = *count;
    const int64_t n = M < (unsigned long long)capacity ? (int64_t)M : capacity;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const uint64_t key = __ldg(keys + i);
#pragma unroll
        for (int p = 0; p < kMaxPasses; ++p)
            if (p < plan.P) atomicAdd(&h[p][(unsigned int)(key >> plan.shift[p]) & plan.mask[p]], 1u);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < plan.P * kRadix; k += blockDim.x) {
        const unsigned int v = (&h[0][0])[k];
        if (v) atomicAdd(hist + k, v);
    }
}

// ------------------------------------------------------------------------------ B3: one radix pass
struct SweepArgs {
    const uint64_t* keys_in; const int32_t* vals_in;
    uint64_t* keys_out; int32_t* vals_out;
    const unsigned long long* count;   // device: number of pairs
    int64_t capacity;
    int shift; unsigned int mask; int pass;
    const unsigned int* hist;        // [256] of this pass
    unsigned long long* status;      // [tiles][256], tag in the high word
    unsigned int* ticket;
};

struct SweepSmem {
    unsigned int warp_hist[kSortWarps][kRadix];
    union {
        unsigned long long keys[kSortTile];
        int vals[kSortTile];
    } x;
    long long goff[kRadix];          // global base of the digit minus its start inside the tile
    unsigned int bin_start[kRadix];
    unsigned char dig[kSortTile];
    unsigned int scan_tmp[kSortWarps];
    unsigned int tile;
};

__global__ void __launch_bounds__(kSortThreads) onesweep_kernel(const SweepArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SweepSmem& sm = *reinterpret_cast<SweepSmem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    const unsigned long long M = *a.count;
    const int64_t n = M < (unsigned long long)a.capacity ? (int64_t)M : a.capacity;
    const int64_t n_tiles = (n + kSortTile - 1) / kSortTile;
    if (tid == 0) sm.tile = atomicAdd(a.ticket, 1u);
    for (int k = tid; k < kSortWarps * kRadix; k += kSortThreads) (&sm.warp_hist[0][0])[k] = 0;
    __syncthreads();
    const int64_t tile = sm.tile;
    if (tile >= n_tiles) return;
    const int64_t base = tile * kSortTile;
    const int valid = (int)((n - base) < kSortTile ? (n - base) : kSortTile);

    // load keys, warp-striped: item j of lane l sits at warp*512 + j*32 + l (order = (j, lane))
    unsigned long long key[kSortItems];
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const int idx = warp * (32 * kSortItems) + j * 32 + lane;
        key[j] = idx < valid ? __ldg(a.keys_in + base + idx) : ~0ull;
    }
    // rank inside the warp, digit by digit, keeping (j, lane) order
    unsigned short rank[kSortItems];
    const unsigned int lt_mask = (1u << lane) - 1u;
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const unsigned int d = (unsigned int)(key[j] >> a.shift) & a.mask;
        const unsigned int peers = __match_any_sync(0xffffffffu, d);
        const int leader = __ffs(peers) - 1;
        unsigned int old = 0;
        if (lane == leader) old = sm.warp_hist[warp][d];
        old = __shfl_sync(0xffffffffu, old, leader);
        rank[j] = (unsigned short)(old + __popc(peers & lt_mask));
        if (lane == leader) sm.warp_hist[warp][d] = old + __popc(peers);
        __syncwarp();
    }
    __syncthreads();
    // thread d owns digit d: per-warp exclusive offsets and the tile's count of this digit
    unsigned int count = 0;
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) {
        const unsigned int c = sm.warp_hist[w][tid];
        sm.warp_hist[w][tid] = count;
        count += c;
    }
    // publish the tile's digit count, then look back for the exclusive prefix over earlier tiles
    const unsigned long long tag_local = ((unsigned long long)(a.pass * 4 + 5)) << 32;
    const unsigned long long tag_incl = ((unsigned long long)(a.pass * 4 + 6)) << 32;
    unsigned long long* my_status = a.status + tile * kRadix + tid;
    st_volatile_u64(my_status, (tile == 0 ? tag_incl : tag_local) | count);
    // exclusive scans over digits: position of the digit inside the tile, and global digit base
    const unsigned int hval = __ldg(a.hist + tid);
    unsigned int inc_c = count, inc_h = hval;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned int oc = __shfl_up_sync(0xffffffffu, inc_c, d);
        const unsigned int oh = __shfl_up_sync(0xffffffffu, inc_h, d);
        if (lane >= d) { inc_c += oc; inc_h += oh; }
    }
    __shared__ unsigned int s_wc[kSortWarps], s_wh[kSortWarps];
    if (lane == 31) { s_wc[warp] = inc_c; s_wh[warp] = inc_h; }
    __syncthreads();
    unsigned int bc = 0, bh = 0;
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w)
        if (w < warp) { bc += s_wc[w]; bh += s_wh[w]; }
    const unsigned int bin_start = bc + inc_c - count;
    const unsigned int digit_base = bh + inc_h - hval;
    unsigned int excl = 0;
    if (tile > 0) {
        int64_t look = tile - 1;
        while (true) {
            unsigned long long st;
            do { st = ld_volatile_u64(a.status + look * kRadix + tid); } while ((st >> 34) != (unsigned long long)(a.pass + 1));
            excl += (unsigned int)st;
            if (((st >> 32) & 3ull) == 2ull) break;
            --look;
        }
        st_volatile_u64(my_status, tag_incl | (unsigned long long)(excl + count));
    }
    sm.bin_start[tid] = bin_start;
    sm.goff[tid] = (long long)digit_base + (long long)excl - (long long)bin_start;
    __syncthreads();
    // keys -> shared memory in sorted order
    unsigned short pos[kSortItems];
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const unsigned int d = (unsigned int)(key[j] >> a.shift) & a.mask;
        pos[j] = (unsigned short)(sm.bin_start[d] + sm.warp_hist[warp][d] + rank[j]);
        sm.x.keys[pos[j]] = key[j];
    }
    // values are fetched while the keys drain
    int val[kSortItems];
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) {
        const int idx = warp * (32 * kSortItems) + j * 32 + lane;
        val[j] = idx < valid ? __ldg(a.vals_in + base + idx) : 0;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kSortItems; ++k) {
        const int p = tid + k * kSortThreads;
        if (p < valid) {
            const unsigned long long kk = sm.x.keys[p];
            const unsigned int d = (unsigned int)(kk >> a.shift) & a.mask;
            sm.dig[p] = (unsigned char)d;
            a.keys_out[sm.goff[d] + p] = kk;
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kSortItems; ++j) sm.x.vals[pos[j]] = val[j];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kSortItems; ++k) {
        const int p = tid + k * kSortThreads;
        if (p < valid) a.vals_out[sm.goff[sm.dig[p]] + p] = sm.x.vals[p];
    }
}

// ------------------------------------------------------------------------------ B3: tile sort
struct TileSweepArgs {
    const unsigned int* keys_in; const int32_t* vals_in;
    unsigned int* keys_out; int32_t* vals_out;
    const unsigned long long* count;   // device: number of records (BinHeader::n_rec)
    int shift; unsigned int mask; int pass;
    const unsigned int* digit_base;    // [BINS] exclusive digit bases of this pass
    unsigned long long* status;        // [tiles][BINS], tag in the high word
    unsigned int* ticket;
};

template <int BITS>
struct TileSweepSmem {
    static constexpr int BINS = 1 << BITS;
    unsigned short warp_hist[kTsWarps][BINS];   // <= 256 items per warp
    unsigned int keys[kTsTile];
    int vals[kTsTile];
    int goff[BINS];                  // global base of the digit minus its start inside the tile
    unsigned int bin_start[BINS];
    unsigned int scan_tmp[kTsWarps];
    unsigned int tile;
};

template <int BITS>
__global__ void __launch_bounds__(kTsThreads, 2) tile_sweep_kernel(const TileSweepArgs a) {
    using Smem = TileSweepSmem<BITS>;
    constexpr int BINS = Smem::BINS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem& sm = *reinterpret_cast<Smem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned int lt_mask = (1u << lane) - 1u;
    const int64_t n = (int64_t)(*a.count);
    const int64_t n_tiles = (n + kTsTile - 1) / kTsTile;
    const unsigned long long tag_local = ((unsigned long long)(a.pass * 4 + 5)) << 32;
    const unsigned long long tag_incl = ((unsigned long long)(a.pass * 4 + 6)) << 32;
    unsigned int dbase = 0;
    if (tid < BINS) dbase = __ldg(a.digit_base + tid);

    while (true) {
        __syncthreads();   // shared memory of the previous tile is no longer read
        if (tid == 0) sm.tile = atomicAdd(a.ticket, 1u);
        for (int k = tid; k < kTsWarps * BINS / 2; k += kTsThreads) reinterpret_cast<unsigned int*>(&sm.warp_hist[0][0])[k] = 0;
        __syncthreads();
        const int64_t tile = sm.tile;
        if (tile >= n_tiles) break;
        const int64_t base = tile * kTsTile;
        const int valid = (int)((n - base) < kTsTile ? (n - base) : kTsTile);

        // load, warp-striped: item j of lane l sits at warp*(32*items) + j*32 + l (order = (j, lane))
        unsigned int key[kTsItems];
        int val[kTsItems];
#pragma unroll
        for (int j = 0; j < kTsItems; ++j) {
            const int idx = warp * (32 * kTsItems) + j * 32 + lane;
            key[j] = idx < valid ? __ldg(a.keys_in + base + idx) : 0xffffffffu;
        }
#pragma unroll
        for (int j = 0; j < kTsItems; ++j) {
            const int idx = warp * (32 * kTsItems) + j * 32 + lane;
            val[j] = idx < valid ? __ldg(a.vals_in + base + idx) : 0;
        }
        // rank inside the warp, digit by digit, keeping (j, lane) order
        unsigned short rank[kTsItems];
#pragma unroll
        for (int j = 0; j < kTsItems; ++j) {
            const unsigned int d = (key[j] >> a.shift) & a.mask;
            const unsigned int peers = __match_any_sync(0xffffffffu, d);
            const int leader = __ffs(peers) - 1;
            unsigned int old = 0;
            if (lane == leader) old = sm.warp_hist[warp][d];
            old = __shfl_sync(0xffffffffu, old, leader);
            rank[j] = (unsigned short)(old + __popc(peers & lt_mask));
            if (lane == leader) sm.warp_hist[warp][d] = (unsigned short)(old + __popc(peers));
            __syncwarp();
        }
        __syncthreads();
        // thread d owns digit d: per-warp exclusive offsets and the tile's count of this digit
        unsigned int count = 0;
        if (tid < BINS) {
#pragma unroll
            for (int w = 0; w < kTsWarps; ++w) {
                const unsigned int c = sm.warp_hist[w][tid];
                sm.warp_hist[w][tid] = (unsigned short)count;
                count += c;
            }
            st_volatile_u64(a.status + tile * BINS + tid, (tile == 0 ? tag_incl : tag_local) | count);
        }
        // exclusive scan over digits: position of the digit inside the tile
        unsigned int inc_c = count;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned int oc = __shfl_up_sync(0xffffffffu, inc_c, d);
            if (lane >= d) inc_c += oc;
        }
        if (lane == 31) sm.scan_tmp[warp] = inc_c;
        __syncthreads();
        if (tid < BINS) {
            unsigned int bc = 0;
#pragma unroll
            for (int w = 0; w < BINS / 32; ++w)
                if (w < warp) bc += sm.scan_tmp[w];
            const unsigned int bin_start = bc + inc_c - count;
            // look back over the earlier tiles for the exclusive prefix of this digit
            unsigned int excl = 0;
            if (tile > 0) {
                int64_t look = tile - 1;
                while (true) {
                    unsigned long long st;
                    do { st = ld_volatile_u64(a.status + look * BINS + tid); } while ((st >> 34) != (unsigned long long)(a.pass + 1));
                    excl += (unsigned int)st;
                    if (((st >> 32) & 3ull) == 2ull) break;
                    --look;
                }
                st_volatile_u64(a.status + tile * BINS + tid, tag_incl | (unsigned long long)(excl + count));
            }
            sm.bin_start[tid] = bin_start;
            sm.goff[tid] = (int)(dbase + excl) - (int)bin_start;
        }
        __syncthreads();
        // records -> shared memory in sorted order
#pragma unroll
        for (int j = 0; j < kTsItems; ++j) {
            const unsigned int d = (key[j] >> a.shift) & a.mask;
            const unsigned int pos = sm.bin_start[d] + sm.warp_hist[warp][d] + rank[j];
            sm.keys[pos] = key[j];
            sm.vals[pos] = val[j];
        }
        __syncthreads();
        // every digit run goes to consecutive global addresses
#pragma unroll
        for (int k = 0; k < kTsItems; ++k) {
            const int p = tid + k * kTsThreads;
            if (p < valid) {
                const unsigned int kk = sm.keys[p];
                const int dst = sm.goff[(kk >> a.shift) & a.mask] + p;
                a.keys_out[dst] = kk;
                a.vals_out[dst] = sm.vals[p];
            }
        }
    }
}

// ------------------------------------------------------------------------------ B4
__global__ void __launch_bounds__(256) ranges_kernel(const unsigned int* __restrict__ tkeys, const unsigned long long* count,
                                                     int64_t* __restrict__ ranges) {
    const int64_t n = (int64_t)(*count);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t t = (int64_t)__ldg(tkeys + i);
        if (i == 0) {
            ranges[2 * t] = 0;
        } else {
            const int64_t tp = (int64_t)__ldg(tkeys + i - 1);
            if (tp != t) {
                ranges[2 * t] = i;
                ranges[2 * tp + 1] = i;
            }
        }
        if (i == n - 1) ranges[2 * t + 1] = n;
    }
}

// optional output: the 64-bit keys of the sorted records
__global__ void __launch_bounds__(256) keys_kernel(const unsigned int* __restrict__ tkeys, const int32_t* __restrict__ vals,
                                                   const float* __restrict__ depths, const unsigned long long* count,
                                                   uint64_t* __restrict__ keys) {
    const int64_t n = (int64_t)(*count);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        keys[i] = ((uint64_t)__ldg(tkeys + i) << 32) | (uint64_t)__float_as_uint(__ldg(depths + __ldg(vals + i)));
}

__global__ void set_count_kernel(unsigned long long* count, unsigned long long n) { *count = n; }

static int sm_count() {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    return sms;
}

// 64-bit radix passes; data starts in (k0, v0) and ping-pongs with (k1, v1)
static int run_sort(const SortPlan& plan, uint64_t* k0, int32_t* v0, uint64_t* k1, int32_t* v1, const unsigned long long* count,
                    unsigned int* tickets, unsigned int* hist, unsigned long long* status, int64_t capacity, cudaStream_t st) {
    if (plan.P == 0) return GS_OK;
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(onesweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SweepSmem)) != cudaSuccess)
            return GS_ERR_CUDA;
        attr_set = true;
    }
    const int sms = sm_count();
    const int64_t tiles = (capacity + kSortTile - 1) / kSortTile;
    const int64_t hist_blocks = tiles < (int64_t)sms * 4 ? tiles : (int64_t)sms * 4;
    hist_kernel<<<(unsigned)hist_blocks, 256, 0, st>>>(k0, count, capacity, plan, hist);
    int rc = launch_status();
    if (rc) return rc;
    for (int p = 0; p < plan.P; ++p) {
        SweepArgs a;
        a.keys_in = (p & 1) ? k1 : k0; a.vals_in = (p & 1) ? v1 : v0;
        a.keys_out = (p & 1) ? k0 : k1; a.vals_out = (p & 1) ? v0 : v1;
        a.count = count; a.capacity = capacity;
        a.shift = plan.shift[p]; a.mask = plan.mask[p]; a.pass = p;
        a.hist = hist + p * kRadix;
        a.status = status;
        a.ticket = tickets + p;
        onesweep_kernel<<<(unsigned)tiles, kSortThreads, sizeof(SweepSmem), st>>>(a);
        rc = launch_status();
        if (rc) return rc;
    }
    return GS_OK;
}

template <int BITS>
static int launch_tile_sweep(const TileSweepArgs& a, int64_t capacity, cudaStream_t st) {
    static int blocks_per_sm = 0;
    const int smem = (int)sizeof(TileSweepSmem<BITS>);
    if (!blocks_per_sm) {
        if (cudaFuncSetAttribute(tile_sweep_kernel<BITS>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return GS_ERR_CUDA;
        int b = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, tile_sweep_kernel<BITS>, kTsThreads, smem) != cudaSuccess || b < 1) return GS_ERR_CUDA;
        blocks_per_sm = b;
    }
    const int64_t tiles = (capacity + kTsTile - 1) / kTsTile;
    const int64_t resident = (int64_t)sm_count() * blocks_per_sm;
    tile_sweep_kernel<BITS><<<(unsigned)(tiles < resident ? tiles : resident), kTsThreads, smem, st>>>(a);
    return launch_status();
}

}  // namespace gs

using namespace gs;

extern "C" int gs_bin_tiles(const gs_config* cfg, int64_t N, int32_t C, const gs_camera* cams, const float* means2d,
                            const float* depths, const int32_t* radii, void* workspace, size_t* workspace_bytes,
                            int64_t capacity_M, uint64_t* isect_keys, int32_t* isect_vals, int64_t* tile_ranges,
                            int64_t* M_dev, int64_t* M_out, void* stream) {
    int rc = check_cfg(cfg);
    if (rc) return rc;
    rc = check_cams(C, cams);
    if (rc) return rc;
    if (N < 0 || capacity_M < 0) return GS_ERR_INVALID_ARGUMENT;
    if ((int64_t)C * N >= (1LL << 31) || capacity_M >= (1LL << 30)) return GS_ERR_UNSUPPORTED;
    const int gx = (cams[0].width + kTile - 1) / kTile, gy = (cams[0].height + kTile - 1) / kTile;
    const int64_t tiles = (int64_t)gx * gy;
    if ((int64_t)C * tiles >= (1LL << 31)) return GS_ERR_UNSUPPORTED;
    const int64_t n_entries = (int64_t)C * N;
    const int64_t cap = capacity_M > 0 ? capacity_M : 1;
    const Workspace w = layout(n_entries, cap);
    if (!workspace) {
        if (!workspace_bytes) return GS_ERR_INVALID_ARGUMENT;
        *workspace_bytes = w.total;
        return GS_OK;
    }
    if (workspace_bytes && *workspace_bytes < w.total) return GS_ERR_INVALID_ARGUMENT;
    if (!isect_vals || !tile_ranges || !aligned(workspace, 256) || !aligned(isect_keys, 8)) return GS_ERR_INVALID_ARGUMENT;
    if (N > 0 && (!means2d || !depths || !radii || !aligned(means2d, 8) || !aligned(radii, 16))) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t st = (cudaStream_t)stream;
    int tile_bits = 1, view_bits = 0;
    while ((1LL << tile_bits) < (int64_t)C * tiles) ++tile_bits;
    while ((1 << view_bits) < C) ++view_bits;
    const SortPlan dplan = make_plan(32 + view_bits, true);
    const TilePlan tplan = make_tile_plan(tile_bits);

    unsigned char* ws = reinterpret_cast<unsigned char*>(workspace);
    BinHeader* hdr = reinterpret_cast<BinHeader*>(ws + w.off_header);
    unsigned int* hist = reinterpret_cast<unsigned int*>(ws + w.off_hist);
    unsigned int* thist = reinterpret_cast<unsigned int*>(ws + w.off_thist);
    uint64_t* ck[2] = {reinterpret_cast<uint64_t*>(ws + w.off_ckeys0), reinterpret_cast<uint64_t*>(ws + w.off_ckeys1)};
    int32_t* cv[2] = {reinterpret_cast<int32_t*>(ws + w.off_cvals0), reinterpret_cast<int32_t*>(ws + w.off_cvals1)};
    unsigned int* tk[2] = {reinterpret_cast<unsigned int*>(ws + w.off_tkeys0), reinterpret_cast<unsigned int*>(ws + w.off_tkeys1)};
    // the tile sort ping-pongs between buffer 0 and 1; the caller's array is the one the last pass writes
    int32_t* tv[2];
    tv[tplan.P & 1] = isect_vals;
    tv[(tplan.P & 1) ^ 1] = reinterpret_cast<int32_t*>(ws + w.off_vals);

    if (cudaMemsetAsync(ws, 0, w.zero_bytes, st) != cudaSuccess) return GS_ERR_CUDA;
    if (cudaMemsetAsync(tile_ranges, 0, (size_t)C * tiles * 2 * sizeof(int64_t), st) != cudaSuccess) return GS_ERR_CUDA;
    const int64_t n_blocks = (n_entries + kScanTile - 1) / kScanTile;
    if (n_blocks > 0) {
        CompactArgs a;
        a.n_entries = n_entries; a.N = N; a.gx = gx; a.gy = gy;
        a.means2d = means2d; a.depths = depths; a.radii = radii;
        a.vcap = w.vcap; a.ckeys = reinterpret_cast<unsigned long long*>(ck[0]); a.cvals = cv[0];
        a.hdr = hdr; a.status = reinterpret_cast<unsigned long long*>(ws + w.off_compact_status);
        a.n_blocks = (unsigned int)n_blocks;
        a.M_dev = reinterpret_cast<unsigned long long*>(M_dev);
        compact_kernel<<<(unsigned)n_blocks, kScanThreads, 0, st>>>(a);
        rc = launch_status();
        if (rc) return rc;
    } else if (M_dev) {
        if (cudaMemsetAsync(M_dev, 0, sizeof(int64_t), st) != cudaSuccess) return GS_ERR_CUDA;
    }
    if (capacity_M > 0 && n_blocks > 0) {
        // depth sort of the visible entries (bits of the fp32 depth, then the view index)
        rc = run_sort(dplan, ck[0], cv[0], ck[1], cv[1], &hdr->V, hdr->sort_ticket, hist,
                      reinterpret_cast<unsigned long long*>(ws + w.off_sort_status), w.vcap, st);
        if (rc) return rc;
        const int32_t* sorted_entries = cv[dplan.P & 1];
        const int sms = sm_count();
        {
            EmitArgs a;
            a.N = N; a.gx = gx; a.gy = gy; a.tiles = (unsigned int)tiles;
            a.means2d = means2d; a.radii = radii; a.cvals = sorted_entries;
            a.capacity = capacity_M; a.tkeys = tk[0]; a.vals = tv[0];
            a.hdr = hdr; a.status = reinterpret_cast<unsigned long long*>(ws + w.off_emit_status);
            a.thist = thist; a.plan = tplan;
            const int64_t eb = (w.vcap + kScanTile - 1) / kScanTile;
            const int64_t resident = (int64_t)sms * 6;
            emit_kernel<<<(unsigned)(eb < resident ? eb : resident), kScanThreads, 0, st>>>(a);
            rc = launch_status();
            if (rc) return rc;
        }
        scan_hist_kernel<<<1, kTsMaxBins, 0, st>>>(thist, tplan.P);
        rc = launch_status();
        if (rc) return rc;
        for (int p = 0; p < tplan.P; ++p) {
            TileSweepArgs a;
            a.keys_in = tk[p & 1]; a.vals_in = tv[p & 1];
            a.keys_out = tk[(p & 1) ^ 1]; a.vals_out = tv[(p & 1) ^ 1];
            a.count = &hdr->n_rec;
            a.shift = tplan.shift[p]; a.mask = tplan.mask[p]; a.pass = p;
            a.digit_base = thist + p * kTsMaxBins;
            a.status = reinterpret_cast<unsigned long long*>(ws + w.off_tsort_status);
            a.ticket = &hdr->tsort_ticket[p];
            rc = tplan.bits == 9 ? launch_tile_sweep<9>(a, capacity_M, st) : launch_tile_sweep<8>(a, capacity_M, st);
            if (rc) return rc;
        }
        const unsigned int* sorted_tiles = tk[tplan.P & 1];
        const int64_t rb = (capacity_M + 255) / 256;
        const unsigned grid = (unsigned)(rb < (int64_t)sms * 8 ? rb : (int64_t)sms * 8);
        ranges_kernel<<<grid, 256, 0, st>>>(sorted_tiles, &hdr->n_rec, tile_ranges);
        rc = launch_status();
        if (rc) return rc;
        if (isect_keys) {
            keys_kernel<<<grid, 256, 0, st>>>(sorted_tiles, isect_vals, depths, &hdr->n_rec, isect_keys);
            rc = launch_status();
            if (rc) return rc;
        }
    }
    if (M_out) {
        unsigned long long m = 0;
        if (cudaMemcpyAsync(&m, &hdr->M, sizeof(m), cudaMemcpyDeviceToHost, st) != cudaSuccess) return GS_ERR_CUDA;
        if (cudaStreamSynchronize(st) != cudaSuccess) return GS_ERR_CUDA;
        *M_out = (int64_t)m;
        if ((int64_t)m > capacity_M) return GS_ERR_CAPACITY;
    }
    return GS_OK;
}

// stand-alone sort: header | histograms | look-back status | ping-pong copy of keys and values
struct SortWorkspace {
    size_t off_count, off_tickets, off_hist, off_status, zero_bytes, off_keys, off_vals, total;
};
static SortWorkspace sort_layout(int64_t n) {
    SortWorkspace w;
    size_t o = 0;
    w.off_count = o; o += 16;
    w.off_tickets = o; o += kMaxPasses * sizeof(unsigned int);
    o = align_up(o, 256);
    w.off_hist = o; o += (size_t)kMaxPasses * kRadix * sizeof(unsigned int);
    o = align_up(o, 256);
    w.off_status = o; o += (size_t)((n + kSortTile - 1) / kSortTile + 1) * kRadix * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.zero_bytes = o;
    w.off_keys = o; o += (size_t)n * sizeof(uint64_t); o = align_up(o, 256);
    w.off_vals = o; o += (size_t)n * sizeof(int32_t); o = align_up(o, 256);
    w.total = o;
    return w;
}

extern "C" int gs_sort_pairs(int64_t n, int32_t end_bit, int32_t skip_bit31, uint64_t* keys, int32_t* vals,
                             void* workspace, size_t* workspace_bytes, void* stream) {
    if (n < 0 || end_bit < 1 || end_bit > 64) return GS_ERR_INVALID_ARGUMENT;
    if (n >= (1LL << 30)) return GS_ERR_UNSUPPORTED;
    const int64_t cap = n > 0 ? n : 1;
    const SortWorkspace w = sort_layout(cap);
    if (!workspace) {
        if (!workspace_bytes) return GS_ERR_INVALID_ARGUMENT;
        *workspace_bytes = w.total;
        return GS_OK;
    }
    if (workspace_bytes && *workspace_bytes < w.total) return GS_ERR_INVALID_ARGUMENT;
    if (n == 0) return GS_OK;
    if (!keys || !vals || !aligned(workspace, 256) || !aligned(keys, 8)) return GS_ERR_INVALID_ARGUMENT;
    const SortPlan plan = make_plan(end_bit, skip_bit31 != 0);
    if (plan.P > kMaxPasses) return GS_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char* ws = reinterpret_cast<unsigned char*>(workspace);
    unsigned long long* count = reinterpret_cast<unsigned long long*>(ws + w.off_count);
    if (cudaMemsetAsync(ws, 0, w.zero_bytes, st) != cudaSuccess) return GS_ERR_CUDA;
    set_count_kernel<<<1, 1, 0, st>>>(count, (unsigned long long)n);
    uint64_t* alt_keys = reinterpret_cast<uint64_t*>(ws + w.off_keys);
    int32_t* alt_vals = reinterpret_cast<int32_t*>(ws + w.off_vals);
    int rc = run_sort(plan, keys, vals, alt_keys, alt_vals, count, reinterpret_cast<unsigned int*>(ws + w.off_tickets),
                      reinterpret_cast<unsigned int*>(ws + w.off_hist), reinterpret_cast<unsigned long long*>(ws + w.off_status), n, st);
    if (rc) return rc;
    if (plan.P & 1) {
        if (cudaMemcpyAsync(keys, alt_keys, (size_t)n * sizeof(uint64_t), cudaMemcpyDeviceToDevice, st) != cudaSuccess) return GS_ERR_CUDA;
        if (cudaMemcpyAsync(vals, alt_vals, (size_t)n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st) != cudaSuccess) return GS_ERR_CUDA;
    }
    return GS_OK;
}
