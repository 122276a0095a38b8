// binning.cu -- tile binning B1..B4 (gs_bin_tiles) and the stand-alone radix sort (gs_sort_pairs).
//
// The result defined by SURVEY.md 8(c) O-B is the list of (tile | depth, entry) records in stable
// key order plus the per-tile ranges.  A stable sort by the 64-bit key (tile << 32 | depth) equals a
// stable sort by depth followed by a stable sort by tile, and only the second one has to touch the M
// records (M is 19..80 times the number V of visible entries).  The per-tile record counts (hence the
// ranges and every digit histogram of the tile sort) do not depend on the order at all: they follow
// from the tile rectangles alone.  So the work is organised as
//
//   compact_kernel      B1a: visible entries (radius > 0, >= 1 tile) in ascending entry order ->
//                       (view << 32 | depth bits, entry), ordered chained scan (decoupled look-back);
//                       each rectangle also adds +1/-1 at its four corners of a per-view difference grid.
//   tile_yscan_kernel,  B4: 2-D prefix sum of the difference grid = records per tile; exclusive scan
//   tile_xscan_kernel,  over the tiles = tile_ranges; the same pass accumulates the digit histograms of
//   tile_ranges_kernel  the tile sort and the total record count M.
//   hist_kernel +       depth sort of the V compacted entries: stable LSD radix sort on the depth bits
//   onesweep_kernel     and the view bits (64-bit keys, 8-bit digits; also serves gs_sort_pairs).
//   offsets_kernel      B1b: per-entry tile counts scanned in DEPTH order -> record offset, first tile
//                       id, rectangle width and entry id (16 bytes per visible entry), plus the first
//                       entry of every chunk (one sort tile, 8192 records) of the record list.
//   tile_sweep_kernel   B2+B3: stable LSD radix sort of the M records on the 32-bit tile id, 2 passes
//                       of 8 or 9 bits for every BASELINE configuration.  The first pass GENERATES its
//                       chunk of records from the entry table (the unsorted record list is never
//                       written to memory), the last pass writes only the values.  Persistent blocks,
//                       per-digit decoupled look-back, ballot-based stable ranking.
//   group_count/scan,   B2+B3 from 4 M records (two-level tile sort, see "two-level tile sort" below): the records that are
//   expand_kernel       generated and sorted by tile_sweep_kernel are (group of 4 x 4 or 8 x 8 tiles, entry); every group then
//                       expands its depth-ordered list into the lists of its tiles, each record written once.
//   keys_kernel         optional: the 64-bit keys (tile << 32 | depth bits) of the sorted records.
//
// Equal (tile, depth) records keep ascending entry order (reading A10) because every step is
// order-preserving: index-ordered compaction, stable depth sort, depth-ordered generation, stable
// tile sort.  The counts V and M live in device memory; no stage needs the host.
#include "common.cuh"

namespace gs {

// ------------------------------------------------------------------------------ workspace layout
struct BinHeader {
    unsigned long long M;          // records the batch needs (sum of tile counts of all visible entries)
    unsigned long long V;          // visible entries (clamped to the compact capacity)
    unsigned long long n_rec;      // records to sort = M, or 0 when M > capacity_M
    unsigned int compact_ticket, xscan_ticket, rscan_ticket, offs_ticket;
    unsigned int sort_ticket[8];   // depth-sort passes
    unsigned int tsort_ticket[4];  // tile-sort passes
    unsigned long long n_crec;     // group records to sort (two-level tile sort) = their number, or 0 when M > capacity_M
};
static_assert(sizeof(BinHeader) == 96, "header size");

constexpr int kRadix = 256;            // depth sort: 8-bit digits
constexpr int kMaxPasses = 8;

constexpr int kScanThreads = 256;      // chained scans: 4 items per thread
constexpr int kScanItems = 4;
constexpr int kScanTile = kScanThreads * kScanItems;

constexpr int kSortThreads = 256;      // depth sort
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSortItems = 16;
constexpr int kSortTile = kSortThreads * kSortItems;

constexpr int kTsThreads = 512;        // tile sort
constexpr int kTsWarps = kTsThreads / 32;
constexpr int kTsItems = 16;
constexpr int kTsTile = kTsThreads * kTsItems;
constexpr int kTsMaxBits = 9;
constexpr int kTsMaxBins = 1 << kTsMaxBits;
constexpr int kTsMaxPasses = 4;
constexpr int kLookWide = 1;                // tile sort: predecessors inspected per look-back round trip (4 and 8 measured: no gain)
// two-level tile sort: groups of 4 x 4 tiles (shorter lists per group, better balance), or 8 x 8 when 4 x 4 gives too many groups
constexpr int64_t kTwoLevelMinRecords = 4 << 20;
constexpr int kMaxGroups = 8192;          // group counters are scanned by one block; beyond this the one-level sort is used

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

// one visible entry in depth order: where its records start, which tiles they are, whose they are
struct __align__(16) EntryRec {
    unsigned int off;      // offset of the entry's first record in the (virtual) unsorted record list
    unsigned int t0;       // tile id of the rectangle's first tile (view * tiles + y0 * gx + x0)
    unsigned int w;        // rectangle width in tiles
    int id;                // entry e = c * N + i
};

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Workspace {
    size_t off_header, off_hist, off_thist, off_tdiff, off_compact_status, off_xscan_status, off_rscan_status, off_offs_status,
        off_sort_status, off_tsort_status, off_cg_count, zero_bytes;
    size_t off_ckeys0, off_ckeys1, off_cvals0, off_cvals1, off_entries, off_chunk_first, off_vmask, off_tkeys0, off_tkeys1, off_vals, off_vals2,
        off_group_start, off_entry_h, total;
    int64_t vcap, cells, n_chunks;
};
static Workspace layout(int64_t n_entries, int64_t capacity, int64_t cells) {
    Workspace w;
    // every visible entry emits >= 1 record, so V <= M; a call that fits capacity has V <= capacity
    w.vcap = n_entries < capacity ? n_entries : capacity;
    if (w.vcap < 1) w.vcap = 1;
    w.cells = cells;
    w.n_chunks = (capacity + kTsTile - 1) / kTsTile;
    size_t o = 0;
    w.off_header = o; o += sizeof(BinHeader);
    o = align_up(o, 256);
    w.off_hist = o; o += (size_t)kMaxPasses * kRadix * sizeof(unsigned int);
    w.off_thist = o; o += (size_t)kTsMaxPasses * kTsMaxBins * sizeof(unsigned int);
    o = align_up(o, 256);
    w.off_tdiff = o; o += (size_t)(cells + kScanTile) * sizeof(int);
    o = align_up(o, 256);
    w.off_compact_status = o; o += (size_t)((n_entries + kScanTile - 1) / kScanTile + 1) * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.off_xscan_status = o; o += (size_t)((cells + kScanTile - 1) / kScanTile + 1) * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.off_rscan_status = o; o += (size_t)((cells + kScanTile - 1) / kScanTile + 1) * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.off_offs_status = o; o += (size_t)((w.vcap + kScanTile - 1) / kScanTile + 1) * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.off_sort_status = o; o += (size_t)((w.vcap + kSortTile - 1) / kSortTile + 1) * kRadix * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.off_tsort_status = o; o += (size_t)(w.n_chunks + 1) * kTsMaxBins * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.off_cg_count = o; o += (size_t)kMaxGroups * sizeof(unsigned int);
    o = align_up(o, 256);
    w.zero_bytes = o;  // everything up to here is cleared at the start of a call
    w.off_ckeys0 = o; o += (size_t)w.vcap * sizeof(uint64_t); o = align_up(o, 256);
    w.off_ckeys1 = o; o += (size_t)w.vcap * sizeof(uint64_t); o = align_up(o, 256);
    w.off_cvals0 = o; o += (size_t)w.vcap * sizeof(int32_t); o = align_up(o, 256);
    w.off_cvals1 = o; o += (size_t)w.vcap * sizeof(int32_t); o = align_up(o, 256);
    w.off_entries = o; o += (size_t)w.vcap * sizeof(EntryRec); o = align_up(o, 256);
    w.off_chunk_first = o; o += (size_t)(w.n_chunks + 2) * sizeof(unsigned int); o = align_up(o, 256);
    w.off_vmask = o; o += (size_t)((n_entries + 31) / 32 + 4) * sizeof(unsigned int); o = align_up(o, 256);   // visibility bits (large inputs)
    w.off_tkeys0 = o; o += (size_t)capacity * sizeof(uint32_t); o = align_up(o, 256);
    w.off_tkeys1 = o; o += (size_t)capacity * sizeof(uint32_t); o = align_up(o, 256);
    w.off_vals = o; o += (size_t)capacity * sizeof(int32_t); o = align_up(o, 256);
    w.off_vals2 = o; o += (size_t)capacity * sizeof(int32_t); o = align_up(o, 256);      // second value buffer of the group sort
    w.off_group_start = o; o += (size_t)(kMaxGroups + 1) * sizeof(unsigned int); o = align_up(o, 256);
    w.off_entry_h = o; o += (size_t)w.vcap * sizeof(unsigned short); o = align_up(o, 256);
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
// prefix, return the exclusive one.  `tile` is the block's position in ticket order.  Sums are taken
// modulo 2^62 (callers that scan signed values truncate the result to 32 bits).
__device__ __forceinline__ unsigned long long chained_scan_lookback(unsigned long long* status, int64_t tile,
                                                                     unsigned long long block_total, int lane) {
    unsigned long long excl = 0;
    if (tile == 0) {
        if (lane == 0) st_volatile_u64(status, kFlagIncl | (block_total & kValMask));
        return 0;
    }
    if (lane == 0) st_volatile_u64(status + tile, kFlagAgg | (block_total & kValMask));
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
    if (lane == 0) st_volatile_u64(status + tile, kFlagIncl | ((excl + block_total) & kValMask));
    return excl;
}

// Block-wide part of an ordered chained scan: every thread passes the sum of its items, gets the
// global exclusive prefix of that sum; `block_total` and `block_excl` are returned to all threads.
struct ChainScanSmem {
    unsigned long long warp_sum[kScanThreads / 32];
    unsigned long long base;
};
__device__ __forceinline__ unsigned long long block_chained_scan(unsigned long long thread_sum, unsigned long long* status, int64_t tile,
                                                                   ChainScanSmem& sm, unsigned long long& block_excl,
                                                                   unsigned long long& block_total) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned long long inc = thread_sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned long long o = shfl_up_u64(inc, d);
        if (lane >= d) inc += o;
    }
    if (lane == 31) sm.warp_sum[warp] = inc;
    __syncthreads();
    unsigned long long wbase = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) {
        if (w < warp) wbase += sm.warp_sum[w];
        total += sm.warp_sum[w];
    }
    if (warp == 0) {
        const unsigned long long excl = chained_scan_lookback(status, tile, total, lane);
        if (lane == 0) sm.base = excl;
    }
    __syncthreads();
    block_excl = sm.base;
    block_total = total;
    return sm.base + wbase + inc - thread_sum;
}

// Block-wide variant of the look-back: all kScanThreads threads inspect one predecessor each per
// round trip (nearest first), so a chain of several thousand in-flight blocks is walked in a handful
// of L2 round trips instead of one per 32 blocks.  Every thread returns the exclusive prefix.
struct WideLookSmem {
    unsigned long long sum[kScanThreads / 32];
    unsigned int has[kScanThreads / 32];
};
__device__ __forceinline__ unsigned long long block_lookback(unsigned long long* status, int64_t tile, unsigned long long block_total,
                                                             WideLookSmem& sm) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tile == 0) {
        if (tid == 0) st_volatile_u64(status, kFlagIncl | (block_total & kValMask));
        return 0;
    }
    if (tid == 0) st_volatile_u64(status + tile, kFlagAgg | (block_total & kValMask));
    unsigned long long excl = 0;
    int64_t look = tile - 1;
    while (true) {
        const int64_t idx = look - tid;
        unsigned long long st = kFlagIncl;   // virtual predecessor of block 0: inclusive 0
        if (idx >= 0) {
            do { st = ld_volatile_u64(status + idx); } while ((st >> 62) == 0);
        }
        const unsigned int incl = __ballot_sync(0xffffffffu, (st >> 62) == 2);
        unsigned long long v = st & kValMask;
        if (incl && lane > __ffs(incl) - 1) v = 0;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v += shfl_u64(v, lane ^ d);
        if (lane == 0) { sm.sum[warp] = v; sm.has[warp] = incl; }
        __syncthreads();
        bool found = false;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w)
            if (!found) { excl += sm.sum[w]; found = sm.has[w] != 0u; }
        if (found) break;
        look -= kScanThreads;
        __syncthreads();   // the round's partial sums have been read
    }
    if (tid == 0) st_volatile_u64(status + tile, kFlagIncl | ((excl + block_total) & kValMask));
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
    int* tdiff;             // [C][gy+1][gx+1] corner differences of the tile rectangles
    BinHeader* hdr;
    unsigned long long* status;
    unsigned int n_blocks;
};

// Warp-striped arrangement: warp w of the block covers 128 * VEC consecutive entries; in iteration
// j lane l holds entries (j * 128 + l * 4 .. + 3) of that span as one 16-byte load, so that the VEC
// loads of a thread are all in flight together (memory-level parallelism) and every warp request is
// 512 contiguous bytes.  Phase 1: visibility (radius > 0 and a non-empty tile rectangle) as one bit
// per entry, corner differences of the rectangle.  Phase 2 (after the ordered chained scan of the
// per-block counts): the visible entries' (view | depth, entry) pairs go to their ranks; ranks keep
// ascending entry order (iteration, lane, component).
template <int VEC>
__global__ void __launch_bounds__(kScanThreads) compact_kernel(const CompactArgs a) {
    pdl_enter();
    constexpr int TILE = kScanThreads * 4 * VEC;
    constexpr int WARPS = kScanThreads / 32;
    __shared__ unsigned int s_ticket;
    __shared__ unsigned int s_warp[WARPS];
    __shared__ WideLookSmem s_look;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_ticket = atomicAdd(&a.hdr->compact_ticket, 1u);
    __syncthreads();
    const int64_t tile = s_ticket;
    const int64_t w0 = tile * TILE + (int64_t)warp * (128 * VEC) + lane * 4;

    int4 rad[VEC];
#pragma unroll
    for (int j = 0; j < VEC; ++j) {
        const int64_t e = w0 + j * 128;
        if (e + 4 <= a.n_entries) {
            rad[j] = __ldg(reinterpret_cast<const int4*>(a.radii + e));
        } else {
            rad[j].x = (e < a.n_entries) ? __ldg(a.radii + e) : 0;
            rad[j].y = (e + 1 < a.n_entries) ? __ldg(a.radii + e + 1) : 0;
            rad[j].z = (e + 2 < a.n_entries) ? __ldg(a.radii + e + 2) : 0;
            rad[j].w = 0;
        }
    }
    const int sx = a.gx + 1, sy = a.gy + 1;
    unsigned int cand = 0;         // bit 4 j + k: entry w0 + 128 j + k has a positive radius
#pragma unroll
    for (int j = 0; j < VEC; ++j)
        cand |= ((rad[j].x > 0 ? 1u : 0u) | (rad[j].y > 0 ? 2u : 0u) | (rad[j].z > 0 ? 4u : 0u) | (rad[j].w > 0 ? 8u : 0u)) << (4 * j);
    // one copy of the per-candidate code (a loop over the set bits, not an unrolled chain: in the
    // large-scene regime a fraction of a per cent of the entries is visible and the instruction
    // footprint of the skip path is what matters); C * N < 2^31, so 32-bit division gives the view
    unsigned int vis = 0;          // candidates with a non-empty tile rectangle
    const unsigned int n32 = (unsigned int)a.N;
    while (cand) {
        const int bit = __ffs(cand) - 1;
        cand &= cand - 1;
        const int64_t e = w0 + (bit >> 2) * 128 + (bit & 3);
        const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + e);
        int x0, x1, y0, y1;
        tile_rect(uv.x, uv.y, __ldg(a.radii + e), a.gx, a.gy, x0, x1, y0, y1);
        if (x1 > x0 && y1 > y0) {
            vis |= 1u << bit;
            int* g = a.tdiff + (int64_t)((unsigned int)e / n32) * ((int64_t)sx * sy);
            atomicAdd(g + y0 * sx + x0, 1);
            atomicAdd(g + y0 * sx + x1, -1);
            atomicAdd(g + y1 * sx + x0, -1);
            atomicAdd(g + y1 * sx + x1, 1);
        }
    }
    // inclusive scan over the lanes of the per-iteration counts (<= 4 each, <= 128 per warp: 8-bit
    // fields, four iterations per word)
    constexpr int WORDS = (VEC + 3) / 4;
    unsigned int inc[WORDS];
#pragma unroll
    for (int q = 0; q < WORDS; ++q) {
        unsigned int c = 0;
#pragma unroll
        for (int j = 4 * q; j < 4 * q + 4 && j < VEC; ++j) c |= (unsigned int)__popc((vis >> (4 * j)) & 15u) << (8 * (j - 4 * q));
        // a field can reach 128 only in lane 31 of the inclusive sum: no carry into the next field
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned int o = __shfl_up_sync(0xffffffffu, c, d);
            if (lane >= d) c += o;
        }
        inc[q] = c;
    }
    // totals of the iterations (lane 31's fields) -> exclusive bases of the iterations inside the warp
    unsigned int iter_base[VEC];
    unsigned int wtotal = 0;
#pragma unroll
    for (int j = 0; j < VEC; ++j) {
        iter_base[j] = wtotal;
        wtotal += (__shfl_sync(0xffffffffu, inc[j / 4], 31) >> (8 * (j % 4))) & 255u;
    }
    if (lane == 0) s_warp[warp] = wtotal;
    __syncthreads();
    unsigned int wbase = 0, btotal = 0;
#pragma unroll
    for (int w = 0; w < WARPS; ++w) {
        if (w < warp) wbase += s_warp[w];
        btotal += s_warp[w];
    }
    const unsigned long long excl = block_lookback(a.status, tile, btotal, s_look);
    if (tid == 0 && tile == (int64_t)a.n_blocks - 1) {
        const unsigned long long V = excl + btotal;
        a.hdr->V = V < (unsigned long long)a.vcap ? V : (unsigned long long)a.vcap;
    }
    if (btotal == 0) return;       // (block-uniform) nothing to write
    const unsigned long long gbase = excl + wbase;
    // exclusive rank of the lane's first visible entry of every iteration, 8-bit fields as above
    unsigned int lane_excl[WORDS];
#pragma unroll
    for (int q = 0; q < WORDS; ++q) {
        unsigned int own = 0;
#pragma unroll
        for (int j = 4 * q; j < 4 * q + 4 && j < VEC; ++j) own |= (unsigned int)__popc((vis >> (4 * j)) & 15u) << (8 * (j - 4 * q));
        lane_excl[q] = inc[q] - own;
    }
    unsigned int m = vis;
    int cur_j = -1;
    unsigned long long pos = 0;
    while (m) {
        const int bit = __ffs(m) - 1;
        m &= m - 1;
        const int j = bit >> 2;
        if (j != cur_j) {
            cur_j = j;
            unsigned int ib = 0, le = 0;
#pragma unroll
            for (int jj = 0; jj < VEC; ++jj)
                if (jj == j) { ib = iter_base[jj]; le = (lane_excl[jj / 4] >> (8 * (jj % 4))) & 255u; }
            pos = gbase + ib + le;
        }
        const int64_t e = w0 + j * 128 + (bit & 3);
        if (pos < (unsigned long long)a.vcap) {
            a.ckeys[pos] = ((unsigned long long)((unsigned int)e / n32) << 32) | (unsigned long long)__float_as_uint(__ldg(a.depths + e));
            a.cvals[pos] = (int)e;
        }
        ++pos;
    }
}

// ---- B1a for large inputs (>= 2^24 entries): two kernels -----------------------------------------
// In the street-scale scenes a fraction of a per cent of the C*N entries is visible, and the fused
// kernel above spends its time in a serial chain per block (ticket -> radii -> candidate gathers ->
// scan -> look-back -> depth gathers).  Here the streaming part carries no ordering at all:
//   visible_kernel       radii -> visibility bit mask (one bit per entry) and the corner differences;
//   compact_mask_kernel  ordered chained scan over the mask (32 768 entries per block, 1/32 of the
//                        bytes), lanes = bits when a mask word is expanded.
constexpr int kMaskVec = 8;                                   // 16-byte loads per thread of visible_kernel
constexpr int kMaskTile = kScanThreads * 4 * kMaskVec;        // 8 192 entries per block
// compact_mask_kernel: WPT mask words per thread -- 16 (512 entries, one ticket per 131 072 entries) for the large sparse inputs
// the mask exists for, 4 when the mask is small (a dense mask then costs at most 128 serial entries per thread)
constexpr int64_t kMaskWideMinWords = 1 << 19;
constexpr int64_t kMaskMinEntries = 1 << 24;                  // measured on B200: fused 50 us vs split 62 us at 10 M entries, 530 vs 265 us at 240 M

__global__ void __launch_bounds__(kScanThreads) visible_kernel(const CompactArgs a, unsigned int* __restrict__ vmask, int64_t n_words) {
    pdl_enter();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t wbase = (int64_t)blockIdx.x * kMaskTile + (int64_t)warp * (128 * kMaskVec);
    const int64_t w0 = wbase + lane * 4;
    int4 rad[kMaskVec];
#pragma unroll
    for (int j = 0; j < kMaskVec; ++j) {
        const int64_t e = w0 + j * 128;
        if (e + 4 <= a.n_entries) {
            rad[j] = __ldg(reinterpret_cast<const int4*>(a.radii + e));
        } else {
            rad[j].x = (e < a.n_entries) ? __ldg(a.radii + e) : 0;
            rad[j].y = (e + 1 < a.n_entries) ? __ldg(a.radii + e + 1) : 0;
            rad[j].z = (e + 2 < a.n_entries) ? __ldg(a.radii + e + 2) : 0;
            rad[j].w = 0;
        }
    }
    const int sx = a.gx + 1, sy = a.gy + 1;
    unsigned int cand = 0;         // bit 4 j + k: entry w0 + 128 j + k has a positive radius
#pragma unroll
    for (int j = 0; j < kMaskVec; ++j)
        cand |= ((rad[j].x > 0 ? 1u : 0u) | (rad[j].y > 0 ? 2u : 0u) | (rad[j].z > 0 ? 4u : 0u) | (rad[j].w > 0 ? 8u : 0u)) << (4 * j);
    unsigned int vis = 0;          // candidates with a non-empty tile rectangle
    const unsigned int n32 = (unsigned int)a.N;
    while (cand) {
        const int bit = __ffs(cand) - 1;
        cand &= cand - 1;
        const int64_t e = w0 + (bit >> 2) * 128 + (bit & 3);
        const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + e);
        int x0, x1, y0, y1;
        tile_rect(uv.x, uv.y, __ldg(a.radii + e), a.gx, a.gy, x0, x1, y0, y1);
        if (x1 > x0 && y1 > y0) {
            vis |= 1u << bit;
            int* g = a.tdiff + (int64_t)((unsigned int)e / n32) * ((int64_t)sx * sy);
            atomicAdd(g + y0 * sx + x0, 1);
            atomicAdd(g + y0 * sx + x1, -1);
            atomicAdd(g + y1 * sx + x0, -1);
            atomicAdd(g + y1 * sx + x1, 1);
        }
    }
    // 8 lanes x 4 bits -> one mask word (bit i of word w = entry 32 w + i)
    const int sh = 4 * (lane & 7);
#pragma unroll
    for (int j = 0; j < kMaskVec; ++j) {
        unsigned int v = ((vis >> (4 * j)) & 15u) << sh;
        v |= __shfl_xor_sync(0xffffffffu, v, 1);
        v |= __shfl_xor_sync(0xffffffffu, v, 2);
        v |= __shfl_xor_sync(0xffffffffu, v, 4);
        const int64_t widx = ((wbase + j * 128) >> 5) + (lane >> 3);
        if ((lane & 7) == 0 && widx < n_words) vmask[widx] = v;
    }
}

// VIEWS = false: `vmask` is the flat mask over the entries e = c N + i written by visible_kernel (which has also added the
// corner differences).  VIEWS = true: `vmask` is the per-view mask [C][wn] written by gs_project_fwd (bit i & 31 of word
// c wn + (i >> 5)); the rectangle corners are added here, from the gathered means2d and radii of the visible entries.
// wn is a multiple of 16 words and a thread owns 16 consecutive words, so a thread's words belong to one view.
// FILL = false (only with VIEWS): the expansion writes nothing but the entry ids; the depth keys and the rectangle corners of
// the compacted entries are produced by entry_fill_kernel, one thread per entry.  When the visible entries are clustered in
// index (a Morton-ordered scene: a few blocks of this kernel own all of them) the gathers then do not hang on the few
// threads whose mask words happen to be full.
template <bool VIEWS, int WPT, bool FILL>
__global__ void __launch_bounds__(kScanThreads) compact_mask_kernel(const CompactArgs a, const unsigned int* __restrict__ vmask, int64_t n_words,
                                                                    int64_t wn) {
    static_assert(FILL || VIEWS, "the split form exists for the caller's per-view mask only");
    pdl_enter();
    __shared__ unsigned int s_ticket;
    __shared__ ChainScanSmem s_scan;
    __shared__ unsigned int s_w[WPT][kScanThreads];     // the thread's words, indexed dynamically in the expansion
    const int tid = threadIdx.x;
    if (tid == 0) s_ticket = atomicAdd(&a.hdr->compact_ticket, 1u);
    __syncthreads();
    const int64_t tile = s_ticket;
    const int64_t wi = tile * (kScanThreads * WPT) + (int64_t)tid * WPT;
    unsigned int cnt = 0, nzw = 0;      // set bits; which of the thread's words are non-zero
#pragma unroll
    for (int v4 = 0; v4 < WPT / 4; ++v4) {
        const int64_t w4 = wi + 4 * v4;
        uint4 v = make_uint4(0u, 0u, 0u, 0u);
        if (w4 + 4 <= n_words) {
            v = __ldg(reinterpret_cast<const uint4*>(vmask + w4));
        } else {
            if (w4 < n_words) v.x = __ldg(vmask + w4);
            if (w4 + 1 < n_words) v.y = __ldg(vmask + w4 + 1);
            if (w4 + 2 < n_words) v.z = __ldg(vmask + w4 + 2);
        }
        s_w[4 * v4][tid] = v.x; s_w[4 * v4 + 1][tid] = v.y; s_w[4 * v4 + 2][tid] = v.z; s_w[4 * v4 + 3][tid] = v.w;
        cnt += (unsigned int)(__popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w));
        nzw |= ((v.x ? 1u : 0u) | (v.y ? 2u : 0u) | (v.z ? 4u : 0u) | (v.w ? 8u : 0u)) << (4 * v4);
    }
    unsigned long long be, bt;
    const unsigned long long pos = block_chained_scan((unsigned long long)cnt, a.status, tile, s_scan, be, bt);
    if (tid == 0 && tile == (int64_t)a.n_blocks - 1) {
        const unsigned long long V = be + bt;
        a.hdr->V = V < (unsigned long long)a.vcap ? V : (unsigned long long)a.vcap;
    }
    if (bt == 0) return;
    // expansion: every thread walks the set bits of its own words, four entries per round so that the gathers of a
    // round are in flight together; its ranks start at the exclusive prefix `pos` (C * N < 2^31: 32-bit ranks)
    const unsigned int n32 = (unsigned int)a.N;
    int64_t e_first = wi << 5;      // entry of bit 0 of this thread's first word
    unsigned int my_view = 0;
    if (VIEWS) {
        my_view = (unsigned int)(wi / wn);
        e_first = (int64_t)my_view * a.N + ((wi - (int64_t)my_view * wn) << 5);
    }
    const int sx = a.gx + 1, sy = a.gy + 1;
    int* const grid = VIEWS ? a.tdiff + (int64_t)my_view * ((int64_t)sx * sy) : nullptr;
    unsigned int r = (unsigned int)pos;
    while (nzw) {
        const int q = __ffs(nzw) - 1;
        nzw &= nzw - 1;
        unsigned int m = s_w[q][tid];
        const int64_t eq = e_first + (q << 5);
        if constexpr (!FILL) {
            while (m) {
                const int64_t e = eq + (__ffs(m) - 1);
                m &= m - 1;
                if ((int64_t)r < a.vcap) {
                    a.cvals[r] = (int)e;
                } else if (VIEWS) {
                    // beyond the compact capacity (the call will report an overflow): the rectangle still counts, M must be exact
                    const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + e);
                    int x0, x1, y0, y1;
                    tile_rect(uv.x, uv.y, __ldg(a.radii + e), a.gx, a.gy, x0, x1, y0, y1);
                    atomicAdd(grid + y0 * sx + x0, 1);
                    atomicAdd(grid + y0 * sx + x1, -1);
                    atomicAdd(grid + y1 * sx + x0, -1);
                    atomicAdd(grid + y1 * sx + x1, 1);
                }
                ++r;
            }
        } else while (m) {
            int64_t e[4];
            bool on[4];
            float dep[4];
            float2 uv[4];
            int rad[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                on[u] = m != 0u;
                e[u] = eq + (on[u] ? __ffs(m) - 1 : 0);
                m &= m - 1;                            // 0 stays 0
                dep[u] = (on[u] && (int64_t)(r + u) < a.vcap) ? __ldg(a.depths + e[u]) : 0.0f;
                if (VIEWS && on[u]) {
                    uv[u] = __ldg(reinterpret_cast<const float2*>(a.means2d) + e[u]);
                    rad[u] = __ldg(a.radii + e[u]);
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (on[u]) {
                    if (VIEWS) {
                        // the rectangle's corner differences (every visible entry, also beyond the compact capacity: M must be exact)
                        int x0, x1, y0, y1;
                        tile_rect(uv[u].x, uv[u].y, rad[u], a.gx, a.gy, x0, x1, y0, y1);
                        atomicAdd(grid + y0 * sx + x0, 1);
                        atomicAdd(grid + y0 * sx + x1, -1);
                        atomicAdd(grid + y1 * sx + x0, -1);
                        atomicAdd(grid + y1 * sx + x1, 1);
                    }
                    if ((int64_t)r < a.vcap) {
                        const unsigned int view = VIEWS ? my_view : (unsigned int)e[u] / n32;
                        a.ckeys[r] = ((unsigned long long)view << 32) | (unsigned long long)__float_as_uint(dep[u]);
                        a.cvals[r] = (int)e[u];
                    }
                    ++r;
                }
        }
    }
}

// Second half of the split compaction: entry r of the compacted list (ids written by compact_mask_kernel<true, WPT, false>)
// gets its (view << 32 | depth bits) key, and its tile rectangle adds +1 / -1 at the four corners of its view's
// difference grid.  One thread per entry, persistent grid.
__global__ void __launch_bounds__(256) entry_fill_kernel(const CompactArgs a) {
    pdl_enter();
    const int64_t V = (int64_t)a.hdr->V;            // already clamped to the compact capacity
    const unsigned int n32 = (unsigned int)a.N;
    const int sx = a.gx + 1, sy = a.gy + 1;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < V; r += (int64_t)gridDim.x * blockDim.x) {
        const unsigned int e = (unsigned int)a.cvals[r];
        const unsigned int view = e / n32;
        const float dep = __ldg(a.depths + e);
        const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + e);
        const int rad = __ldg(a.radii + e);
        a.ckeys[r] = ((unsigned long long)view << 32) | (unsigned long long)__float_as_uint(dep);
        int x0, x1, y0, y1;
        tile_rect(uv.x, uv.y, rad, a.gx, a.gy, x0, x1, y0, y1);
        int* const grid = a.tdiff + (int64_t)view * ((int64_t)sx * sy);
        atomicAdd(grid + y0 * sx + x0, 1);
        atomicAdd(grid + y0 * sx + x1, -1);
        atomicAdd(grid + y1 * sx + x0, -1);
        atomicAdd(grid + y1 * sx + x1, 1);
    }
}

// ------------------------------------------------------------------------------ B4: counts, ranges, histograms
// column prefix sums of the difference grid.  A block owns 32 adjacent columns (lane = column, coalesced rows); its 8
// warps split the rows, every thread loads its rows at once (one memory round trip instead of one per 8 rows of a
// column-serial walk: 13.6 -> 4.4 us on the 4K grid), and the warps' column totals are combined through shared memory.
constexpr int kYscanWarps = 8;
constexpr int kYscanMaxRows = 40;          // rows per thread held in registers; taller grids walk in slabs of 8 x 40 rows
__global__ void __launch_bounds__(32 * kYscanWarps) tile_yscan_kernel(int* __restrict__ tdiff, int C, int gx, int gy) {
    pdl_enter();
    __shared__ int s_tot[kYscanWarps][32];
    const int sx = gx + 1, sy = gy + 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int col = blockIdx.x * 32 + lane;
    const bool live = col < C * sx;
    const int view = live ? col / sx : 0, x = live ? col - view * sx : 0;
    int* p = tdiff + (int64_t)view * sx * sy + x;
    int carry = 0;                                             // column sum of the slabs above
    for (int y0 = 0; y0 < sy; y0 += kYscanWarps * kYscanMaxRows) {
        const int slab = min(sy - y0, kYscanWarps * kYscanMaxRows);
        const int per = (slab + kYscanWarps - 1) / kYscanWarps;   // rows per warp (block-uniform)
        const int r0 = y0 + warp * per, r1 = min(r0 + per, y0 + slab);
        int v[kYscanMaxRows];
#pragma unroll
        for (int k = 0; k < kYscanMaxRows; ++k) v[k] = (live && r0 + k < r1) ? p[(int64_t)(r0 + k) * sx] : 0;
        int acc = 0;
#pragma unroll
        for (int k = 0; k < kYscanMaxRows; ++k) { acc += v[k]; v[k] = acc; }
        s_tot[warp][lane] = acc;
        __syncthreads();
        int base = carry, all = 0;
#pragma unroll
        for (int w = 0; w < kYscanWarps; ++w) {
            const int t = s_tot[w][lane];
            if (w < warp) base += t;
            all += t;
        }
        carry += all;
#pragma unroll
        for (int k = 0; k < kYscanMaxRows; ++k)
            if (live && r0 + k < r1) p[(int64_t)(r0 + k) * sx] = v[k] + base;
        __syncthreads();
    }
}

// inclusive prefix sum of the flattened grid (every padded row sums to zero, so the running sum at a
// cell is the number of rectangles covering that tile); in place
__global__ void __launch_bounds__(kScanThreads) tile_xscan_kernel(int* __restrict__ tdiff, int64_t cells, BinHeader* hdr,
                                                                  unsigned long long* status) {
    pdl_enter();
    __shared__ unsigned int s_ticket;
    __shared__ ChainScanSmem s_scan;
    const int tid = threadIdx.x;
    if (tid == 0) s_ticket = atomicAdd(&hdr->xscan_ticket, 1u);
    __syncthreads();
    const int64_t tile = s_ticket;
    const int64_t i0 = tile * kScanTile + (int64_t)tid * kScanItems;
    // the array is padded to a multiple of the scan tile (zeros), so vector access is always in bounds
    int4 v = *reinterpret_cast<const int4*>(tdiff + i0);
    const int s = v.x + v.y + v.z + v.w;
    unsigned long long be, bt;
    const unsigned int excl = (unsigned int)block_chained_scan((unsigned long long)(long long)s, status, tile, s_scan, be, bt);
    v.x += (int)excl; v.y += v.x; v.z += v.y; v.w += v.z;
    if (i0 < cells) *reinterpret_cast<int4*>(tdiff + i0) = v;
}

// exclusive scan of the per-tile counts -> tile_ranges; digit histograms of the tile sort; M
struct RangesArgs {
    const int* tcount;          // flattened padded grid after both scans
    int64_t cells;
    int32_t C, gx, gy;
    int64_t capacity;
    int64_t* ranges;            // [C * gx * gy][2]
    unsigned int* thist;        // [P][kTsMaxBins]
    TilePlan plan;
    BinHeader* hdr;
    unsigned long long* status;
    unsigned int n_blocks;
    unsigned long long* M_dev;
};

__global__ void __launch_bounds__(kScanThreads) tile_ranges_kernel(const RangesArgs a) {
    pdl_enter();
    __shared__ unsigned int s_ticket;
    __shared__ ChainScanSmem s_scan;
    __shared__ unsigned int s_hist[kTsMaxPasses * kTsMaxBins];
    const int tid = threadIdx.x;
    if (tid == 0) s_ticket = atomicAdd(&a.hdr->rscan_ticket, 1u);
    for (int k = tid; k < a.plan.P * kTsMaxBins; k += kScanThreads) s_hist[k] = 0;
    __syncthreads();
    const int64_t tile = s_ticket;
    const int64_t i0 = tile * kScanTile + (int64_t)tid * kScanItems;
    const int sx = a.gx + 1, sy = a.gy + 1;
    const int4 v4 = *reinterpret_cast<const int4*>(a.tcount + i0);
    int cnt[kScanItems] = {v4.x, v4.y, v4.z, v4.w};
    long long tid_of[kScanItems];
    unsigned long long sum = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        const int64_t i = i0 + k;
        tid_of[k] = -1;
        if (i < a.cells) {
            const int64_t row = i / sx;
            const int x = (int)(i - row * sx);
            const int64_t view = row / sy;
            const int y = (int)(row - view * sy);
            if (x < a.gx && y < a.gy) tid_of[k] = (view * a.gy + y) * a.gx + x;
        }
        if (tid_of[k] < 0) cnt[k] = 0;
        sum += (unsigned long long)cnt[k];
    }
    unsigned long long be, bt;
    unsigned long long start = block_chained_scan(sum, a.status, tile, s_scan, be, bt);
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (tid_of[k] >= 0) {
            const bool some = cnt[k] > 0;
            a.ranges[2 * tid_of[k]] = some ? (int64_t)start : 0;
            a.ranges[2 * tid_of[k] + 1] = some ? (int64_t)(start + cnt[k]) : 0;
            if (some) {
                const unsigned int t = (unsigned int)tid_of[k];
#pragma unroll
                for (int p = 0; p < kTsMaxPasses; ++p)
                    if (p < a.plan.P) atomicAdd(&s_hist[p * kTsMaxBins + ((t >> a.plan.shift[p]) & a.plan.mask[p])], (unsigned int)cnt[k]);
            }
            start += cnt[k];
        }
    }
    if (tid == 0 && tile == (int64_t)a.n_blocks - 1) {
        const unsigned long long M = be + bt;
        a.hdr->M = M;
        a.hdr->n_rec = M <= (unsigned long long)a.capacity ? M : 0ull;
        if (a.M_dev) *a.M_dev = M;
    }
    __syncthreads();
    for (int k = tid; k < a.plan.P * kTsMaxBins; k += kScanThreads) {
        const unsigned int v = s_hist[k];
        if (v) atomicAdd(a.thist + k, v);   // wraps only when M >= 2^32, i.e. far beyond the capacity limit
    }
}

// exclusive scan of the tile-sort digit histograms (one block); when the records do not fit the
// capacity nothing is sorted, so every range is cleared ("outputs incomplete, nothing out of bounds")
__global__ void __launch_bounds__(kTsMaxBins) scan_hist_kernel(unsigned int* thist, int P, const BinHeader* hdr, int64_t capacity,
                                                               int64_t* ranges, int64_t n_ranges) {
    pdl_enter();
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
    if (hdr->M > (unsigned long long)capacity)
        for (int64_t k = tid; k < 2 * n_ranges; k += kTsMaxBins) ranges[k] = 0;
}

// ------------------------------------------------------------------------------ B1b: entry table in depth order
struct OffsetsArgs {
    int64_t N;
    int32_t gx, gy;
    unsigned int tiles;            // gx * gy
    const float* means2d; const int32_t* radii;
    const int32_t* cvals;          // visible entries in (view, depth, entry) order
    EntryRec* entries;
    unsigned int* chunk_first;     // [n_chunks]: entry holding record c * kTsTile
    int64_t n_chunks;
    BinHeader* hdr;
    unsigned long long* status;
    // two-level tile sort: the records generated from the entry table are (GROUP of 8 x 8 tiles, entry) instead of (tile, entry)
    int32_t coarse, gshift, ggx, ggy;   // gshift: log2 of the group side in tiles (2 or 3)
    unsigned int groups;           // ggx * ggy
    unsigned short* entry_h;       // [V] height of the entry's group rectangle (group mode)
};

__global__ void __launch_bounds__(kScanThreads) offsets_kernel(const OffsetsArgs a) {
    pdl_enter();
    __shared__ unsigned int s_ticket;
    __shared__ ChainScanSmem s_scan;
    const int tid = threadIdx.x;
    const unsigned long long V = a.hdr->V;
    const int64_t n_blocks = (int64_t)((V + kScanTile - 1) / kScanTile);
    if ((int64_t)blockIdx.x >= n_blocks) return;     // (the grid is sized for the capacity; only n_blocks blocks take a ticket)
    if (tid == 0) s_ticket = atomicAdd(&a.hdr->offs_ticket, 1u);
    __syncthreads();
    const int64_t tile = s_ticket;
    if (tile >= n_blocks) return;
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
            const unsigned int view = (unsigned int)((int64_t)id[k] / a.N);
            if (a.coarse) {
                // the rectangle of 8 x 8-tile groups the tile rectangle touches; one count per group record
                const int side = 1 << a.gshift;
                x0 >>= a.gshift; y0 >>= a.gshift;
                x1 = (x1 + side - 1) >> a.gshift; y1 = (y1 + side - 1) >> a.gshift;
                ww[k] = (unsigned int)(x1 - x0);
                cnt[k] = ww[k] * (unsigned int)(y1 - y0);
                t0[k] = view * a.groups + (unsigned int)y0 * (unsigned int)a.ggx + (unsigned int)x0;
            } else {
                ww[k] = (unsigned int)(x1 - x0);
                cnt[k] = ww[k] * (unsigned int)(y1 - y0);
                t0[k] = view * a.tiles + (unsigned int)y0 * (unsigned int)a.gx + (unsigned int)x0;
            }
            t_tiles += cnt[k];
        }
    }
    unsigned long long be, bt;
    unsigned long long off = block_chained_scan(t_tiles, a.status, tile, s_scan, be, bt);
    if (a.coarse && tid == 0 && tile == n_blocks - 1) a.hdr->n_crec = a.hdr->n_rec ? be + bt : 0ull;   // (n_rec = 0: the records do not fit)
#pragma unroll
    for (int k = 0; k < kScanItems; ++k)
        if (id[k] >= 0) {
            EntryRec r;
            r.off = (unsigned int)off; r.t0 = t0[k]; r.w = ww[k]; r.id = id[k];
            a.entries[j0 + k] = r;
            if (a.coarse) a.entry_h[j0 + k] = (unsigned short)(cnt[k] / ww[k]);
            // chunks whose first record lies inside this entry
            const unsigned long long c_lo = (off + kTsTile - 1) / kTsTile, c_hi = (off + cnt[k] - 1) / kTsTile;
            for (unsigned long long c = c_lo; c <= c_hi && c < (unsigned long long)a.n_chunks; ++c) a.chunk_first[c] = (unsigned int)(j0 + k);
            off += cnt[k];
        }
}

// ------------------------------------------------------------------------------ two-level tile sort
// The M (tile, entry) records are 19..80 per visible entry, and sorting them by tile id was the largest part of the
// binning (two radix passes over M records, ballot ranking: issue bound).  Instead the records that are GENERATED AND SORTED
// are (group of 4 x 4 or 8 x 8 tiles, entry): 2.4..10 per entry.  Each group then expands its own list (already in depth
// order) into the lists of its 16 or 64 tiles: a warp owns one tile row of the group, lanes = 32 consecutive entries of the
// group's list, and one ballot per tile gives the entries that cover it in list order, i.e. their positions behind the
// tile's running base.  The per-tile ranges come from the difference grid as before, so every record is written once,
// straight to its final place.
// records per group: persistent blocks with a private shared-memory histogram over the groups (a few thousand counters; the
// same counts as global atomics from the chained-scan kernel cost 0.8 ms on the room scene: 7 M atomics on 2 040 addresses)
__global__ void __launch_bounds__(256) group_count_kernel(const EntryRec* __restrict__ entries, const unsigned short* __restrict__ entry_h,
                                                          const BinHeader* hdr, int ggx, int n_groups, unsigned int* __restrict__ cg_count) {
    pdl_enter();
    extern __shared__ unsigned int s_cnt[];
    for (int k = threadIdx.x; k < n_groups; k += blockDim.x) s_cnt[k] = 0;
    __syncthreads();
    const int64_t V = (int64_t)hdr->V;
    // four entries per thread and round, so that four loads are in flight (a thread walks V / (grid * 256) entries).
    // (Tried: one contiguous range of the (view, depth)-ordered entries per block, so that a block touches one view's
    // counters: 25 -> 40 us on city -- neighbouring entries hit the same few counters.)
    const int64_t step = (int64_t)gridDim.x * blockDim.x;
    for (int64_t j0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j0 < V; j0 += 4 * step) {
        uint4 raw[4];
        unsigned int h[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int64_t j = j0 + u * step;
            const bool on = j < V;
            raw[u] = on ? __ldg(reinterpret_cast<const uint4*>(entries + j)) : make_uint4(0u, 0u, 0u, 0u);
            h[u] = on ? (unsigned int)__ldg(entry_h + j) : 0u;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const unsigned int t0 = raw[u].y, w = raw[u].z;
            for (unsigned int y = 0; y < h[u]; ++y)
                for (unsigned int x = 0; x < w; ++x) atomicAdd(&s_cnt[t0 + y * (unsigned int)ggx + x], 1u);
        }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < n_groups; k += blockDim.x) {
        const unsigned int v = s_cnt[k];
        if (v) atomicAdd(cg_count + k, v);
    }
}

// inclusive scan over the 512 threads of a block (warp shuffles + one shared-memory hop); `total` = sum over the block
__device__ __forceinline__ unsigned int block512_inclusive_scan(unsigned int v, unsigned int* s_warp /*[16]*/, unsigned int& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned int o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
    }
    __syncthreads();                 // s_warp free again
    if (lane == 31) s_warp[warp] = v;
    __syncthreads();
    unsigned int base = 0, all = 0;
#pragma unroll
    for (int w = 0; w < 16; ++w) {
        const unsigned int t = s_warp[w];
        if (w < warp) base += t;
        all += t;
    }
    total = all;
    return v + base;
}

__global__ void __launch_bounds__(512) group_scan_kernel(const unsigned int* __restrict__ cg_count, int n_groups, unsigned int* __restrict__ group_start,
                                                         unsigned int* thist, const TilePlan plan) {
    pdl_enter();
    __shared__ unsigned int s_hist[kTsMaxPasses * kTsMaxBins];
    __shared__ unsigned int s_warp[16];
    const int tid = threadIdx.x;
    for (int k = tid; k < plan.P * kTsMaxBins; k += 512) s_hist[k] = 0;
    __syncthreads();
    // exclusive scan of the group counts (16 consecutive groups per thread, n_groups <= 8192) -> group_start
    constexpr int PER = kMaxGroups / 512;
    static_assert(kTsMaxBins == 512, "one histogram bin per thread");
    unsigned int c[PER], sum = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int g = tid * PER + k;
        c[k] = g < n_groups ? cg_count[g] : 0u;
        sum += c[k];
    }
    // digit histograms of the group sort: consecutive groups share the high digits, so a thread adds runs, not single groups
    for (int p = 0; p < plan.P; ++p) {
        unsigned int run = 0, bin = 0xffffffffu;
#pragma unroll
        for (int k = 0; k < PER; ++k) {
            const unsigned int d = (((unsigned int)(tid * PER + k)) >> plan.shift[p]) & plan.mask[p];
            if (d != bin) {
                if (run) atomicAdd(&s_hist[p * kTsMaxBins + bin], run);
                bin = d; run = 0;
            }
            run += c[k];
        }
        if (run) atomicAdd(&s_hist[p * kTsMaxBins + bin], run);
    }
    unsigned int total;
    unsigned int run = block512_inclusive_scan(sum, s_warp, total) - sum;
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int g = tid * PER + k;
        if (g < n_groups) group_start[g] = run;
        run += c[k];
    }
    if (tid == 511) group_start[n_groups] = total;
    // exclusive scans of the digit histograms of the group sort (the barriers inside the scan order the atomics above)
    for (int p = 0; p < plan.P; ++p) {
        __syncthreads();
        const unsigned int v = s_hist[p * kTsMaxBins + tid];
        thist[p * kTsMaxBins + tid] = block512_inclusive_scan(v, s_warp, total) - v;
    }
}

struct ExpandArgs {
    int64_t N;
    int32_t gx, gy, ggx;
    unsigned int tiles, groups;      // gx * gy, ggx * ggy
    const float* means2d; const int32_t* radii;
    const int32_t* cvals;            // group records (entry ids) in (group, depth, entry) order
    const unsigned int* group_start; // [C * groups + 1]
    const int64_t* ranges;           // per-tile ranges (from the difference grid)
    int32_t* vals_out;
    unsigned int* tkeys_out;         // optional: tile id of every record (for the 64-bit keys)
    const BinHeader* hdr;
};

constexpr int kExpChunk = 256;       // group records staged per round

template <int SHIFT>
__global__ void __launch_bounds__(32 << SHIFT) expand_kernel(const ExpandArgs a) {
    pdl_enter();
    constexpr int SIDE = 1 << SHIFT;               // tiles per group side; one warp per tile row of the group
    constexpr int THREADS = 32 * SIDE;
    constexpr int PER = kExpChunk / THREADS;       // entries staged per thread and round
    __shared__ unsigned int s_rect[2][kExpChunk];   // x0 | x1 << 4 | y0 << 8 | y1 << 12, tile coordinates relative to the group (0..SIDE)
    __shared__ int s_id[2][kExpChunk];
    __shared__ unsigned int s_base[SIDE * SIDE];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (a.hdr->n_crec == 0) return;                 // nothing was sorted (no records, or they do not fit: every range is [0, 0))
    const unsigned int g = blockIdx.x;
    const unsigned int begin = __ldg(a.group_start + g), end = __ldg(a.group_start + g + 1);
    if (begin == end) return;
    const unsigned int view = g / a.groups, gl = g - view * a.groups;
    const int tx0 = (int)(gl % (unsigned int)a.ggx) << SHIFT, ty0 = (int)(gl / (unsigned int)a.ggx) << SHIFT;
    if (tid < SIDE * SIDE) {
        const int tx = tx0 + (tid & (SIDE - 1)), ty = ty0 + (tid >> SHIFT);
        s_base[tid] = (tx < a.gx && ty < a.gy) ? (unsigned int)__ldg(a.ranges + 2 * ((int64_t)view * a.tiles + (int64_t)ty * a.gx + tx)) : 0u;
    }
    // software pipeline: list entries two rounds ahead, their (mean, radius) one round ahead
    const unsigned int n = end - begin;
    const unsigned int rounds = (n + kExpChunk - 1) / kExpChunk;
    int id1[PER], id2[PER];
    float2 uv[PER];
    int rad[PER];
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        const unsigned int k = q * THREADS + tid;
        id1[q] = (k < n) ? __ldg(a.cvals + begin + k) : -1;
        id2[q] = (kExpChunk + k < n) ? __ldg(a.cvals + begin + kExpChunk + k) : -1;
    }
#pragma unroll
    for (int q = 0; q < PER; ++q) {
        uv[q] = make_float2(0.f, 0.f); rad[q] = 0;
        if (id1[q] >= 0) { uv[q] = __ldg(reinterpret_cast<const float2*>(a.means2d) + id1[q]); rad[q] = __ldg(a.radii + id1[q]); }
    }
    auto put = [&](int buf, int slot, int id, float2 m, int r) {
        unsigned int packed = 0;
        if (id >= 0) {
            int x0, x1, y0, y1;
            tile_rect(m.x, m.y, r, a.gx, a.gy, x0, x1, y0, y1);
            x0 = clampi(x0 - tx0, 0, SIDE); x1 = clampi(x1 - tx0, 0, SIDE);
            y0 = clampi(y0 - ty0, 0, SIDE); y1 = clampi(y1 - ty0, 0, SIDE);
            packed = (unsigned int)x0 | ((unsigned int)x1 << 4) | ((unsigned int)y0 << 8) | ((unsigned int)y1 << 12);
        }
        s_rect[buf][slot] = packed;
        s_id[buf][slot] = id;
    };
#pragma unroll
    for (int q = 0; q < PER; ++q) put(0, q * THREADS + tid, id1[q], uv[q], rad[q]);
    __syncthreads();
    unsigned int base[SIDE];
#pragma unroll
    for (int x = 0; x < SIDE; ++x) base[x] = s_base[warp * SIDE + x];
    const unsigned int lt = (1u << lane) - 1u;
    const unsigned int tile_row = view * a.tiles + (unsigned int)(ty0 + warp) * (unsigned int)a.gx + (unsigned int)tx0;
    for (unsigned int rd = 0; rd < rounds; ++rd) {
        const int buf = rd & 1;
        // gathers of the next round, list entries of the one after
        int idn[PER];
        float2 uvn[PER];
        int radn[PER];
#pragma unroll
        for (int q = 0; q < PER; ++q) {
            idn[q] = id2[q];
            uvn[q] = make_float2(0.f, 0.f); radn[q] = 0;
            if (idn[q] >= 0) { uvn[q] = __ldg(reinterpret_cast<const float2*>(a.means2d) + idn[q]); radn[q] = __ldg(a.radii + idn[q]); }
            const unsigned int k2 = (rd + 2) * kExpChunk + q * THREADS + tid;
            id2[q] = (k2 < n) ? __ldg(a.cvals + begin + k2) : -1;
        }
        // this warp's tile row against the staged entries, 32 at a time in list order
        const int n_sub = min(kExpChunk / 32, (int)((n - rd * kExpChunk + 31) / 32));
#pragma unroll 1
        for (int sub = 0; sub < n_sub; ++sub) {
            const unsigned int r = s_rect[buf][sub * 32 + lane];
            const unsigned int x0 = r & 15u, x1 = (r >> 4) & 15u, y0 = (r >> 8) & 15u, y1 = r >> 12;
            const bool rowok = (y0 <= (unsigned int)warp) && ((unsigned int)warp < y1);
            if (!__any_sync(0xffffffffu, rowok)) continue;
            const int id = s_id[buf][sub * 32 + lane];
#pragma unroll
            for (int x = 0; x < SIDE; ++x) {
                const bool cov = rowok && (x0 <= (unsigned int)x) && ((unsigned int)x < x1);
                const unsigned int m = __ballot_sync(0xffffffffu, cov);
                if (cov) {
                    const unsigned int pos = base[x] + (unsigned int)__popc(m & lt);
                    a.vals_out[pos] = id;
                    if (a.tkeys_out) a.tkeys_out[pos] = tile_row + (unsigned int)x;
                }
                base[x] += (unsigned int)__popc(m);
            }
        }
        if (rd + 1 < rounds) {
#pragma unroll
            for (int q = 0; q < PER; ++q) put(buf ^ 1, q * THREADS + tid, idn[q], uvn[q], radn[q]);
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------ histograms
__global__ void __launch_bounds__(256) hist_kernel(const uint64_t* __restrict__ keys, const unsigned long long* count, int64_t capacity,
                                                   const SortPlan plan, unsigned int* __restrict__ hist) {
    pdl_enter();
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
    pdl_enter();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SweepSmem& sm = *reinterpret_cast<SweepSmem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    const unsigned long long M = *a.count;
    const int64_t n = M < (unsigned long long)a.capacity ? (int64_t)M : a.capacity;
    const int64_t n_tiles = (n + kSortTile - 1) / kSortTile;
    if ((int64_t)blockIdx.x >= n_tiles) return;       // (the grid is sized for the capacity; only n_tiles blocks take a ticket)
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
        // Look-back, kDepthLookWide predecessors per round: when the blocks of a pass start together (a few hundred tiles, one
        // wave) every tile has published its local count long before any inclusive prefix exists, and the walk over the
        // predecessors is a chain of dependent L2 reads; with several status words in flight per round it costs a
        // quarter of the round trips (depth sort pass of object, 196 tiles: 22.7 -> 20.3 us).
        constexpr int kDepthLookWide = 4;
        int64_t look = tile - 1;
        bool done = false;
        while (!done) {
            unsigned long long st[kDepthLookWide];
#pragma unroll
            for (int u = 0; u < kDepthLookWide; ++u) {
                const int64_t t = look - u;
                st[u] = t >= 0 ? ld_volatile_u64(a.status + t * kRadix + tid) : 0ull;
            }
#pragma unroll
            for (int u = 0; u < kDepthLookWide; ++u) {
                if (done) break;
                if ((st[u] >> 34) != (unsigned long long)(a.pass + 1)) break;      // not published yet: poll again from here
                excl += (unsigned int)st[u];
                --look;
                if (((st[u] >> 32) & 3ull) == 2ull) done = true;
            }
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

// ------------------------------------------------------------------------------ B2 + B3: tile sort
struct TileSweepArgs {
    const unsigned int* keys_in; const int32_t* vals_in;   // unused by the generating pass
    unsigned int* keys_out; int32_t* vals_out;               // keys_out may be NULL in the last pass
    const unsigned long long* count;   // device: number of records (BinHeader::n_rec)
    int shift; unsigned int mask; int pass;
    const unsigned int* digit_base;    // [BINS] exclusive digit bases of this pass
    unsigned long long* status;        // [tiles][BINS], tag in the high word
    unsigned int* ticket;
    // generating pass
    const EntryRec* entries; const unsigned int* chunk_first; const unsigned long long* n_entries; int32_t gx;
};

template <int BITS>
struct TileSweepSmem {
    static constexpr int BINS = 1 << BITS;
    unsigned short warp_hist[kTsWarps][BINS];   // <= 32 * kTsItems items per warp
    unsigned int keys[kTsTile + kTsTile / 32];   // + padding of the generating pass (one word per 32: the blocked
    int vals[kTsTile + kTsTile / 32];            //   writes, 16 words apart between lanes, stay conflict-free)
    int goff[BINS];                  // global base of the digit minus its start inside the tile
    unsigned int bin_start[BINS];
    unsigned short head[kTsTile];    // generating pass: 1 + (entry - first entry) at the entry's first record
    unsigned int scan_tmp[kTsWarps];
    unsigned int tile, next_tile;
};

template <int BITS, bool GEN>
__global__ void __launch_bounds__(kTsThreads, 2) tile_sweep_kernel(const TileSweepArgs a) {
    pdl_enter();
    using Smem = TileSweepSmem<BITS>;
    constexpr int BINS = Smem::BINS;
    static_assert(kTsItems % 8 == 0, "blocked generation reads 8 heads per vector");
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
    if (tid == 0) sm.next_tile = atomicAdd(a.ticket, 1u);

    while (true) {
        __syncthreads();   // shared memory of the previous tile is no longer read; next_tile is visible
        const int64_t tile = sm.next_tile;
        if (tile >= n_tiles) break;
        for (int k = tid; k < kTsWarps * BINS / 2; k += kTsThreads) reinterpret_cast<unsigned int*>(&sm.warp_hist[0][0])[k] = 0;
        if (GEN)
            for (int k = tid; k < kTsTile / 2; k += kTsThreads) reinterpret_cast<unsigned int*>(sm.head)[k] = 0;
        const int64_t base = tile * kTsTile;
        const int valid = (int)((n - base) < kTsTile ? (n - base) : kTsTile);
        __syncthreads();

        unsigned int key[kTsItems];
        int val[kTsItems];
        if (GEN) {
            // ---- generate the chunk's records from the entry table (depth order)
            const unsigned int j0 = __ldg(a.chunk_first + tile);
            const unsigned int j1 = (tile + 1 < n_tiles) ? __ldg(a.chunk_first + tile + 1) : (unsigned int)(*a.n_entries - 1);
            for (unsigned int j = j0 + tid; j <= j1; j += kTsThreads) {
                const unsigned int off = __ldg(&a.entries[j].off);
                const long long slot = (long long)off - (long long)base;
                if (slot < valid) sm.head[slot > 0 ? slot : 0] = (unsigned short)(j - j0 + 1);
            }
            __syncthreads();
            // blocked arrangement: thread owns kTsItems consecutive records; running maximum of the heads
            unsigned int e_rel[kTsItems];
            unsigned int run = 0;
#pragma unroll
            for (int v8 = 0; v8 < kTsItems / 8; ++v8) {
                const uint4 h = *reinterpret_cast<const uint4*>(&sm.head[tid * kTsItems + v8 * 8]);
                const unsigned int hw[4] = {h.x, h.y, h.z, h.w};
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    run = max(run, hw[q] & 0xffffu); e_rel[v8 * 8 + 2 * q] = run;
                    run = max(run, hw[q] >> 16); e_rel[v8 * 8 + 2 * q + 1] = run;
                }
            }
            unsigned int inc = run;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) inc = max(inc, __shfl_up_sync(0xffffffffu, inc, d));
            if (lane == 31) sm.scan_tmp[warp] = inc;
            unsigned int carry = __shfl_up_sync(0xffffffffu, inc, 1);
            if (lane == 0) carry = 0;
            __syncthreads();
#pragma unroll
            for (int w = 0; w < kTsWarps; ++w)
                if (w < warp) carry = max(carry, sm.scan_tmp[w]);
            unsigned int cur = 0xffffffffu;
            EntryRec en;
            en.off = 0; en.t0 = 0; en.w = 1; en.id = 0;
            float inv_w = 1.0f;
#pragma unroll
            for (int k = 0; k < kTsItems; ++k) {
                const int p = tid * kTsItems + k;
                if (p < valid) {
                    const unsigned int er = max(carry, e_rel[k]);   // >= 1: record 0 of the chunk always has a head
                    if (er != cur) {
                        cur = er;
                        const uint4 raw = __ldg(reinterpret_cast<const uint4*>(a.entries + (j0 + er - 1)));
                        en.off = raw.x; en.t0 = raw.y; en.w = raw.z; en.id = (int)raw.w;
                        inv_w = __frcp_rn((float)en.w);
                    }
                    // record index inside the entry -> (row, column) of its tile rectangle: reciprocal
                    // estimate, then an exact fix-up
                    const unsigned int kk = (unsigned int)(base + p) - en.off;
                    unsigned int ry = (unsigned int)(((float)kk + 0.5f) * inv_w);
                    int rx = (int)(kk - ry * en.w);
                    if (rx < 0) { --ry; rx += (int)en.w; }
                    else if (rx >= (int)en.w) { ++ry; rx -= (int)en.w; }
                    sm.keys[p + (p >> 5)] = en.t0 + ry * (unsigned int)a.gx + (unsigned int)rx;
                    sm.vals[p + (p >> 5)] = en.id;
                }
            }
            __syncthreads();
            // warp-striped arrangement for the ranking: item j of lane l is record warp*32*items + j*32 + l
#pragma unroll
            for (int j = 0; j < kTsItems; ++j) {
                const int idx = warp * (32 * kTsItems) + j * 32 + lane;
                key[j] = idx < valid ? sm.keys[idx + (idx >> 5)] : 0xffffffffu;
                val[j] = idx < valid ? sm.vals[idx + (idx >> 5)] : 0;
            }
        } else {
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
        }
        // ---- rank inside the warp, digit by digit, keeping (j, lane) order
        unsigned short rank[kTsItems];
#pragma unroll
        for (int j = 0; j < kTsItems; ++j) {
            const unsigned int d = (key[j] >> a.shift) & a.mask;
            // lanes with the same digit, from one ballot per digit bit (MATCH.ANY occupies the ADU pipe
            // for ~64 cycles per warp instruction on sm_100a; ballots go through the ALU path)
            unsigned int peers = 0xffffffffu;
#pragma unroll
            for (int b = 0; b < BITS; ++b) {
                const bool bit = (d >> b) & 1u;
                const unsigned int m = __ballot_sync(0xffffffffu, bit);
                peers &= bit ? m : ~m;
            }
            const int leader = __ffs(peers) - 1;
            unsigned int old = 0;
            if (lane == leader) old = sm.warp_hist[warp][d];
            old = __shfl_sync(0xffffffffu, old, leader);
            rank[j] = (unsigned short)(old + __popc(peers & lt_mask));
            if (lane == leader) sm.warp_hist[warp][d] = (unsigned short)(old + __popc(peers));
            __syncwarp();
        }
        __syncthreads();   // (also: every thread has read its generated records out of sm.keys / sm.vals)
        // ---- thread d owns digit d: per-warp exclusive offsets and the tile's count of this digit
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
        unsigned int bin_start = 0;
        if (tid < BINS) {
            unsigned int bc = 0;
#pragma unroll
            for (int w = 0; w < BINS / 32; ++w)
                if (w < warp) bc += sm.scan_tmp[w];
            bin_start = bc + inc_c - count;
            sm.bin_start[tid] = bin_start;
        }
        __syncthreads();
        // ---- records -> shared memory in sorted order (needs only tile-local offsets); the look-back comes after
        //      it, so that the predecessors have had this time to publish their counts
#pragma unroll
        for (int j = 0; j < kTsItems; ++j) {
            const unsigned int d = (key[j] >> a.shift) & a.mask;
            const unsigned int pos = sm.bin_start[d] + sm.warp_hist[warp][d] + rank[j];
            sm.keys[pos] = key[j];
            sm.vals[pos] = val[j];
        }
        if (tid < BINS) {
            // look back over the earlier tiles for the exclusive prefix of this digit
            // (kLookWide predecessors are read per round trip: the walk is latency bound)
            unsigned int excl = 0;
            if (tile > 0) {
                int64_t look = tile - 1;
                bool done = false;
                while (!done) {
                    unsigned long long st[kLookWide];
#pragma unroll
                    for (int q = 0; q < kLookWide; ++q)
                        st[q] = (look - q >= 0) ? ld_volatile_u64(a.status + (look - q) * BINS + tid) : 0ull;
#pragma unroll
                    for (int q = 0; q < kLookWide; ++q) {
                        if (!done) {
                            while ((st[q] >> 34) != (unsigned long long)(a.pass + 1)) st[q] = ld_volatile_u64(a.status + (look - q) * BINS + tid);
                            excl += (unsigned int)st[q];
                            done = ((st[q] >> 32) & 3ull) == 2ull;   // tile 0 always publishes an inclusive prefix
                        }
                    }
                    look -= kLookWide;
                }
                st_volatile_u64(a.status + tile * BINS + tid, tag_incl | (unsigned long long)(excl + count));
            }
            sm.goff[tid] = (int)(dbase + excl) - (int)bin_start;
        }
        __syncthreads();
        // ---- every digit run goes to consecutive global addresses
#pragma unroll
        for (int k = 0; k < kTsItems; ++k) {
            const int p = tid + k * kTsThreads;
            if (p < valid) {
                const unsigned int kk = sm.keys[p];
                const int dst = sm.goff[(kk >> a.shift) & a.mask] + p;
                if (a.keys_out) a.keys_out[dst] = kk;
                a.vals_out[dst] = sm.vals[p];
            }
        }
        // The next ticket is claimed only now, when the block is free: tiles then START in ticket order, and a
        // look-back rarely meets a predecessor that has not published yet (claiming it early, while this tile was
        // processed, cost 22 % of bin_tiles on the room scene).
        if (tid == 0) sm.next_tile = atomicAdd(a.ticket, 1u);
    }
}

// optional output: the 64-bit keys of the sorted records
__global__ void __launch_bounds__(256) keys_kernel(const unsigned int* __restrict__ tkeys, const int32_t* __restrict__ vals,
                                                   const float* __restrict__ depths, const unsigned long long* count,
                                                   uint64_t* __restrict__ keys) {
    pdl_enter();
    const int64_t n = (int64_t)(*count);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        keys[i] = ((uint64_t)__ldg(tkeys + i) << 32) | (uint64_t)__float_as_uint(__ldg(depths + __ldg(vals + i)));
}

__global__ void set_count_kernel(unsigned long long* count, unsigned long long n) { pdl_enter(); *count = n; }

// 64-bit radix passes; data starts in (k0, v0) and ping-pongs with (k1, v1)
static int run_sort(const SortPlan& plan, uint64_t* k0, int32_t* v0, uint64_t* k1, int32_t* v1, const unsigned long long* count,
                    unsigned int* tickets, unsigned int* hist, unsigned long long* status, int64_t capacity, cudaStream_t st) {
    if (plan.P == 0) return GS_OK;
    if (int rc0 = ensure_smem(onesweep_kernel, 1, (int)sizeof(SweepSmem))) return rc0;
    const int sms = sm_count();
    const int64_t tiles = (capacity + kSortTile - 1) / kSortTile;
    const int64_t hist_blocks = tiles < (int64_t)sms * 4 ? tiles : (int64_t)sms * 4;
    launch_chained(hist_kernel, dim3((unsigned)hist_blocks), dim3(256), (size_t)(0), st, k0, count, capacity, plan, hist);
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
        launch_chained(onesweep_kernel, dim3((unsigned)tiles), dim3(kSortThreads), (size_t)(sizeof(SweepSmem)), st, a);
        rc = launch_status();
        if (rc) return rc;
    }
    return GS_OK;
}

template <int BITS, bool GEN>
static int launch_tile_sweep(const TileSweepArgs& a, int64_t capacity, cudaStream_t st) {
    const int smem = (int)sizeof(TileSweepSmem<BITS>);
    constexpr int slot = 2 + (BITS == 9 ? 2 : 0) + (GEN ? 1 : 0);
    if (int rc0 = ensure_smem(tile_sweep_kernel<BITS, GEN>, slot, smem)) return rc0;
    DeviceCache& dc = device_cache();
    if (!dc.occ[slot]) {
        int b = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, tile_sweep_kernel<BITS, GEN>, kTsThreads, smem) != cudaSuccess || b < 1) return GS_ERR_CUDA;
        dc.occ[slot] = b;
    }
    const int64_t tiles = (capacity + kTsTile - 1) / kTsTile;
    const int64_t resident = (int64_t)dc.sms * dc.occ[slot];
    launch_chained(tile_sweep_kernel<BITS, GEN>, dim3((unsigned)(tiles < resident ? tiles : resident)), dim3(kTsThreads), (size_t)(smem), st, a);
    return launch_status();
}

}  // namespace gs

using namespace gs;

extern "C" int gs_bin_tiles(const gs_config* cfg, int64_t N, int32_t C, const gs_camera* cams, const float* means2d,
                            const float* depths, const int32_t* radii, const uint32_t* vis_mask, void* workspace, size_t* workspace_bytes,
                            int64_t capacity_M, uint64_t* isect_keys, int32_t* isect_vals, int64_t* tile_ranges,
                            int64_t* M_dev, int64_t* M_out, int32_t tile_sort, void* stream) {
    int rc = check_cfg(cfg);
    if (rc) return rc;
    rc = check_cams(C, cams);
    if (rc) return rc;
    if (N < 0 || capacity_M < 0) return GS_ERR_INVALID_ARGUMENT;
    if ((int64_t)C * N >= (1LL << 31) || capacity_M >= (1LL << 30)) return GS_ERR_UNSUPPORTED;
    const int gx = (cams[0].width + kTile - 1) / kTile, gy = (cams[0].height + kTile - 1) / kTile;
    const int64_t tiles = (int64_t)gx * gy;
    const int64_t cells = (int64_t)C * (gx + 1) * (gy + 1);
    if ((int64_t)C * tiles >= (1LL << 31) || cells >= (1LL << 31)) return GS_ERR_UNSUPPORTED;
    const int64_t n_entries = (int64_t)C * N;
    const int64_t cap = capacity_M > 0 ? capacity_M : 1;
    const Workspace w = layout(n_entries, cap, cells);
    if (!workspace) {
        if (!workspace_bytes) return GS_ERR_INVALID_ARGUMENT;
        *workspace_bytes = w.total;
        return GS_OK;
    }
    if (workspace_bytes && *workspace_bytes < w.total) return GS_ERR_INVALID_ARGUMENT;
    if (!isect_vals || !tile_ranges || !aligned(workspace, 256) || !aligned(isect_keys, 8)) return GS_ERR_INVALID_ARGUMENT;
    if (N > 0 && (!means2d || !depths || !radii || !aligned(means2d, 8) || !aligned(radii, 16) || !aligned(vis_mask, 16))) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t st = (cudaStream_t)stream;
    int tile_bits = 1, view_bits = 0;
    while ((1LL << tile_bits) < (int64_t)C * tiles) ++tile_bits;
    while ((1 << view_bits) < C) ++view_bits;
    const SortPlan dplan = make_plan(32 + view_bits, true);
    // two-level tile sort (groups of 8 x 8 tiles) unless the batch has more groups than one block scans
    // Group side: 4 x 4 tiles (shorter lists per group, better balance between the expanding blocks), 8 x 8 when the lists
    // are long anyway (>= 512 records per tile expected: fewer group records to sort) or when 4 x 4 gives too many groups.
    // Small batches keep the one-level sort: below 4 M records its two passes cost less than the extra launches.
    // Measured on B200 (bin_tiles, one-level / 4 x 4 / 8 x 8): room (124 M records) 2.44 / 0.93 / 0.86 ms, object (14.7 M)
    // 0.49 / 0.39 / 0.44, city (9 M) 0.41 / 0.37 / 0.38, block (2 M) 0.21 / 0.25 / 0.30.
    if (tile_sort < 0 || tile_sort > 3) return GS_ERR_INVALID_ARGUMENT;
    int gshift = 2;
    if ((int64_t)C * ((gx + 3) >> 2) * ((gy + 3) >> 2) > kMaxGroups || capacity_M >= 512 * (int64_t)C * tiles) gshift = 3;
    if (tile_sort == GS_TILE_SORT_GROUPS_4 || tile_sort == GS_TILE_SORT_GROUPS_8) gshift = tile_sort == GS_TILE_SORT_GROUPS_4 ? 2 : 3;
    const int ggx = (gx + (1 << gshift) - 1) >> gshift, ggy = (gy + (1 << gshift) - 1) >> gshift;
    const int64_t n_groups = (int64_t)C * ggx * ggy;
    if (tile_sort >= GS_TILE_SORT_GROUPS_4 && n_groups > kMaxGroups) return GS_ERR_UNSUPPORTED;
    const bool two_level = tile_sort == GS_TILE_SORT_AUTO ? (n_groups <= kMaxGroups && capacity_M >= kTwoLevelMinRecords)
                                                          : tile_sort != GS_TILE_SORT_ONE_LEVEL;
    int group_bits = 1;
    while ((1LL << group_bits) < n_groups) ++group_bits;
    const TilePlan tplan = make_tile_plan(two_level ? group_bits : tile_bits);
    const int sms = sm_count();

    unsigned char* ws = reinterpret_cast<unsigned char*>(workspace);
    BinHeader* hdr = reinterpret_cast<BinHeader*>(ws + w.off_header);
    unsigned int* hist = reinterpret_cast<unsigned int*>(ws + w.off_hist);
    unsigned int* thist = reinterpret_cast<unsigned int*>(ws + w.off_thist);
    int* tdiff = reinterpret_cast<int*>(ws + w.off_tdiff);
    auto status_at = [&](size_t off) { return reinterpret_cast<unsigned long long*>(ws + off); };
    uint64_t* ck[2] = {reinterpret_cast<uint64_t*>(ws + w.off_ckeys0), reinterpret_cast<uint64_t*>(ws + w.off_ckeys1)};
    int32_t* cv[2] = {reinterpret_cast<int32_t*>(ws + w.off_cvals0), reinterpret_cast<int32_t*>(ws + w.off_cvals1)};
    unsigned int* tk[2] = {reinterpret_cast<unsigned int*>(ws + w.off_tkeys0), reinterpret_cast<unsigned int*>(ws + w.off_tkeys1)};
    // pass p writes buffer (p + 1) & 1; the caller's array is the one the last pass writes
    int32_t* tv[2];
    tv[tplan.P & 1] = isect_vals;
    tv[(tplan.P & 1) ^ 1] = reinterpret_cast<int32_t*>(ws + w.off_vals);

    if (cudaMemsetAsync(ws, 0, w.zero_bytes, st) != cudaSuccess) return GS_ERR_CUDA;
    // compaction tile: the largest of 1, 2, 4, 8 x 1024 entries per block that still gives 8 blocks per SM
    int cvec = 8;
    while (cvec > 1 && n_entries < (int64_t)kScanTile * cvec * sms * 8) cvec >>= 1;
    const int64_t n_blocks = (n_entries + (int64_t)kScanTile * cvec - 1) / ((int64_t)kScanTile * cvec);
    if (n_blocks > 0) {
        CompactArgs a;
        a.n_entries = n_entries; a.N = N; a.gx = gx; a.gy = gy;
        a.means2d = means2d; a.depths = depths; a.radii = radii;
        a.vcap = w.vcap; a.ckeys = reinterpret_cast<unsigned long long*>(ck[0]); a.cvals = cv[0];
        a.tdiff = tdiff;
        a.hdr = hdr; a.status = status_at(w.off_compact_status);
        a.n_blocks = (unsigned int)n_blocks;
        if (vis_mask) {
            // the caller's visibility mask (written by gs_project_fwd): ordered scan over the mask, no pass over the radii
            const int64_t wn = GS_VIS_WORDS(N), n_words = (int64_t)C * wn;
            if (n_words >= kMaskWideMinWords) {
                a.n_blocks = (unsigned int)((n_words + kScanThreads * 16 - 1) / (kScanThreads * 16));
                launch_chained(compact_mask_kernel<true, 16, false>, dim3(a.n_blocks), dim3(kScanThreads), (size_t)(0), st, a, vis_mask, n_words, wn);
            } else {
                a.n_blocks = (unsigned int)((n_words + kScanThreads * 4 - 1) / (kScanThreads * 4));
                launch_chained(compact_mask_kernel<true, 4, false>, dim3(a.n_blocks), dim3(kScanThreads), (size_t)(0), st, a, vis_mask, n_words, wn);
            }
            rc = launch_status();
            if (rc) return rc;
            const int64_t fb = (w.vcap + 255) / 256;
            launch_chained(entry_fill_kernel, dim3((unsigned)(fb < (int64_t)sms * 8 ? (fb > 0 ? fb : 1) : (int64_t)sms * 8)), dim3(256), (size_t)(0), st, a);
        } else if (n_entries >= kMaskMinEntries) {
            // large inputs: streaming visibility mask, then the ordered scan over the mask
            unsigned int* vmask = reinterpret_cast<unsigned int*>(ws + w.off_vmask);
            const int64_t n_words = (n_entries + 31) / 32;
            launch_chained(visible_kernel, dim3((unsigned)((n_entries + kMaskTile - 1) / kMaskTile)), dim3(kScanThreads), (size_t)(0), st, a, vmask, n_words);
            rc = launch_status();
            if (rc) return rc;
            a.n_blocks = (unsigned int)((n_words + kScanThreads * 16 - 1) / (kScanThreads * 16));
            launch_chained(compact_mask_kernel<false, 16, true>, dim3(a.n_blocks), dim3(kScanThreads), (size_t)(0), st, a, vmask, n_words, 0);
        } else switch (cvec) {
            case 8: launch_chained(compact_kernel<8>, dim3((unsigned)n_blocks), dim3(kScanThreads), (size_t)(0), st, a); break;
            case 4: launch_chained(compact_kernel<4>, dim3((unsigned)n_blocks), dim3(kScanThreads), (size_t)(0), st, a); break;
            case 2: launch_chained(compact_kernel<2>, dim3((unsigned)n_blocks), dim3(kScanThreads), (size_t)(0), st, a); break;
            default: launch_chained(compact_kernel<1>, dim3((unsigned)n_blocks), dim3(kScanThreads), (size_t)(0), st, a); break;
        }
        rc = launch_status();
        if (rc) return rc;
    }
    // records per tile -> ranges, digit histograms, M
    {
        const int cols = C * (gx + 1);
        launch_chained(tile_yscan_kernel, dim3((cols + 31) / 32), dim3(32 * kYscanWarps), (size_t)(0), st, tdiff, C, gx, gy);
        rc = launch_status();
        if (rc) return rc;
        const unsigned int cb = (unsigned int)((cells + kScanTile - 1) / kScanTile);
        launch_chained(tile_xscan_kernel, dim3(cb), dim3(kScanThreads), (size_t)(0), st, tdiff, cells, hdr, status_at(w.off_xscan_status));
        rc = launch_status();
        if (rc) return rc;
        RangesArgs a;
        a.tcount = tdiff; a.cells = cells; a.C = C; a.gx = gx; a.gy = gy; a.capacity = capacity_M;
        a.ranges = tile_ranges; a.thist = thist; a.plan = tplan; a.hdr = hdr; a.status = status_at(w.off_rscan_status);
        if (two_level) a.plan.P = 0;      // (the digit histograms of the group sort come from the group counts, below)
        a.n_blocks = cb; a.M_dev = reinterpret_cast<unsigned long long*>(M_dev);
        launch_chained(tile_ranges_kernel, dim3(cb), dim3(kScanThreads), (size_t)(0), st, a);
        rc = launch_status();
        if (rc) return rc;
        launch_chained(scan_hist_kernel, dim3(1), dim3(kTsMaxBins), (size_t)(0), st, thist, two_level ? 0 : tplan.P, hdr, capacity_M, tile_ranges, (int64_t)C * tiles);
        rc = launch_status();
        if (rc) return rc;
    }
    if (capacity_M > 0 && n_blocks > 0) {
        // depth sort of the visible entries (bits of the fp32 depth, then the view index)
        rc = run_sort(dplan, ck[0], cv[0], ck[1], cv[1], &hdr->V, hdr->sort_ticket, hist, status_at(w.off_sort_status), w.vcap, st);
        if (rc) return rc;
        const int32_t* sorted_entries = cv[dplan.P & 1];
        EntryRec* entries = reinterpret_cast<EntryRec*>(ws + w.off_entries);
        unsigned int* chunk_first = reinterpret_cast<unsigned int*>(ws + w.off_chunk_first);
        {
            OffsetsArgs a;
            a.N = N; a.gx = gx; a.gy = gy; a.tiles = (unsigned int)tiles;
            a.means2d = means2d; a.radii = radii; a.cvals = sorted_entries;
            a.entries = entries; a.chunk_first = chunk_first; a.n_chunks = w.n_chunks;
            a.hdr = hdr; a.status = status_at(w.off_offs_status);
            a.coarse = two_level ? 1 : 0; a.gshift = gshift; a.ggx = ggx; a.ggy = ggy; a.groups = (unsigned int)(ggx * ggy);
            a.entry_h = reinterpret_cast<unsigned short*>(ws + w.off_entry_h);
            launch_chained(offsets_kernel, dim3((unsigned)((w.vcap + kScanTile - 1) / kScanTile)), dim3(kScanThreads), (size_t)(0), st, a);
            rc = launch_status();
            if (rc) return rc;
        }
        unsigned int* group_start = reinterpret_cast<unsigned int*>(ws + w.off_group_start);
        int32_t* gv[2] = {reinterpret_cast<int32_t*>(ws + w.off_vals), reinterpret_cast<int32_t*>(ws + w.off_vals2)};
        if (two_level) {
            const int64_t vb = (w.vcap + 255) / 256;
            launch_chained(group_count_kernel, dim3((unsigned)(vb < 2 * sms ? vb : 2 * sms)), dim3(256), (size_t)((size_t)n_groups * sizeof(unsigned int)), st, 
                entries, reinterpret_cast<const unsigned short*>(ws + w.off_entry_h), hdr, ggx, (int)n_groups,
                reinterpret_cast<unsigned int*>(ws + w.off_cg_count));
            rc = launch_status();
            if (rc) return rc;
            launch_chained(group_scan_kernel, dim3(1), dim3(512), (size_t)(0), st, reinterpret_cast<const unsigned int*>(ws + w.off_cg_count), (int)n_groups, group_start, thist, tplan);
            rc = launch_status();
            if (rc) return rc;
        }
        for (int p = 0; p < tplan.P; ++p) {
            const bool last = p == tplan.P - 1;
            TileSweepArgs a;
            a.keys_in = tk[p & 1]; a.vals_in = two_level ? gv[p & 1] : tv[p & 1];
            a.keys_out = (last && (two_level || !isect_keys)) ? nullptr : tk[(p & 1) ^ 1];
            a.vals_out = two_level ? gv[(p & 1) ^ 1] : tv[(p & 1) ^ 1];
            a.count = two_level ? &hdr->n_crec : &hdr->n_rec;
            a.shift = tplan.shift[p]; a.mask = tplan.mask[p]; a.pass = p;
            a.digit_base = thist + p * kTsMaxBins;
            a.status = status_at(w.off_tsort_status);
            a.ticket = &hdr->tsort_ticket[p];
            a.entries = entries; a.chunk_first = chunk_first; a.n_entries = &hdr->V; a.gx = two_level ? ggx : gx;
            if (p == 0)
                rc = tplan.bits == 9 ? launch_tile_sweep<9, true>(a, capacity_M, st) : launch_tile_sweep<8, true>(a, capacity_M, st);
            else
                rc = tplan.bits == 9 ? launch_tile_sweep<9, false>(a, capacity_M, st) : launch_tile_sweep<8, false>(a, capacity_M, st);
            if (rc) return rc;
        }
        const unsigned int* sorted_tile_ids = tk[tplan.P & 1];
        if (two_level) {
            // every group expands its (depth-ordered) list into the lists of its 64 tiles
            ExpandArgs a;
            a.N = N; a.gx = gx; a.gy = gy; a.ggx = ggx; a.tiles = (unsigned int)tiles; a.groups = (unsigned int)(ggx * ggy);
            a.means2d = means2d; a.radii = radii; a.cvals = gv[tplan.P & 1]; a.group_start = group_start; a.ranges = tile_ranges;
            a.vals_out = isect_vals; a.tkeys_out = isect_keys ? tk[0] : nullptr; a.hdr = hdr;
            if (gshift == 2) launch_chained(expand_kernel<2>, dim3((unsigned)n_groups), dim3(128), (size_t)(0), st, a);
            else launch_chained(expand_kernel<3>, dim3((unsigned)n_groups), dim3(256), (size_t)(0), st, a);
            rc = launch_status();
            if (rc) return rc;
            sorted_tile_ids = tk[0];
        }
        if (isect_keys) {
            const int64_t rb = (capacity_M + 255) / 256;
            const unsigned grid = (unsigned)(rb < (int64_t)sms * 8 ? rb : (int64_t)sms * 8);
            launch_chained(keys_kernel, dim3(grid), dim3(256), (size_t)(0), st, sorted_tile_ids, isect_vals, depths, &hdr->n_rec, isect_keys);
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
    launch_chained(set_count_kernel, dim3(1), dim3(1), (size_t)(0), st, count, (unsigned long long)n);
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

// ---------------------------------------------------------------------------------------------
// gs_sort_pairs_static: gs_sort_pairs for callers that cannot allocate.  The workspace of the stand-alone sort (count,
// pass tickets, digit histograms, look-back status words, ping-pong copy of keys and values: sort_layout) is a file-scope
// device array sized for GS_SORT_STATIC_MAX_N pairs.  In HOST code the array's name is only a stand-in for the symbol, not
// a device address: the address is resolved once per device with cudaGetSymbolAddress (below) and that pointer is what
// the kernels receive.  One array per device, shared by every call and never cleared between calls: the call zeroes the
// words that must start at zero, exactly as gs_sort_pairs does with its workspace; calls that overlap on the GPU race.
namespace gs {
constexpr size_t static_align(size_t x) { return (x + 255) / 256 * 256; }
constexpr size_t kSortStaticBytes =
    static_align(16 + kMaxPasses * sizeof(unsigned int)) +                                                     // count, tickets
    static_align((size_t)kMaxPasses * kRadix * sizeof(unsigned int)) +                                         // histograms
    static_align((size_t)((GS_SORT_STATIC_MAX_N + kSortTile - 1) / kSortTile + 1) * kRadix * sizeof(unsigned long long)) +   // status
    static_align((size_t)GS_SORT_STATIC_MAX_N * sizeof(uint64_t)) + static_align((size_t)GS_SORT_STATIC_MAX_N * sizeof(int32_t));
static __device__ __align__(256) unsigned char g_sort_static_scratch[kSortStaticBytes];

// device address of the scratch array on the current device (resolved once per device; idempotent, so concurrent first
// calls are harmless)
static int sort_static_scratch(unsigned char** out) {
    static unsigned char* ptr[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return GS_ERR_CUDA;
    if (dev < 0 || dev >= 64) return GS_ERR_UNSUPPORTED;
    if (!ptr[dev]) {
        unsigned char* p = nullptr;
        if (cudaGetSymbolAddress((void**)&p, g_sort_static_scratch) != cudaSuccess || !p) {
            cudaGetLastError();
            return GS_ERR_CUDA;
        }
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return GS_OK;
}
}  // namespace gs

extern "C" int gs_sort_pairs_static(int64_t n, int32_t end_bit, int32_t skip_bit31, uint64_t* keys, int32_t* vals, void* stream) {
    if (n < 0 || end_bit < 1 || end_bit > 64) return GS_ERR_INVALID_ARGUMENT;
    if (n > (int64_t)GS_SORT_STATIC_MAX_N) return GS_ERR_UNSUPPORTED;        // beyond the static scratch: nothing is launched
    unsigned char* ws = nullptr;
    if (int rc = sort_static_scratch(&ws)) return rc;
    if (n == 0) return GS_OK;
    if (!keys || !vals || !aligned(keys, 8) || !aligned(vals, 4)) return GS_ERR_INVALID_ARGUMENT;
    const SortWorkspace w = sort_layout(n);
    if (w.total > kSortStaticBytes) return GS_ERR_UNSUPPORTED;               // (cannot happen for n <= GS_SORT_STATIC_MAX_N)
    const SortPlan plan = make_plan(end_bit, skip_bit31 != 0);
    if (plan.P > kMaxPasses) return GS_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* count = reinterpret_cast<unsigned long long*>(ws + w.off_count);
    // what must start at zero: count, tickets, histograms, status words (the previous call's values are still there)
    if (cudaMemsetAsync(ws, 0, w.zero_bytes, st) != cudaSuccess) return GS_ERR_CUDA;
    launch_chained(set_count_kernel, dim3(1), dim3(1), (size_t)(0), st, count, (unsigned long long)n);
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
