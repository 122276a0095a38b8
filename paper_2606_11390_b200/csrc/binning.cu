// binning.cu -- tile binning B1..B4 (gs_bin_tiles) and the stand-alone radix sort (gs_sort_pairs).
//
//   emit_kernel      B1+B2 fused: single-pass chained scan (decoupled look-back) of the per-entry
//                    tile counts, then a warp-cooperative emit of (key, value) records.  The ordered
//                    look-back replaces an unordered atomic counter so that equal keys keep ascending
//                    entry order (SURVEY.md 8(c) reading A10) and the values are bit-exact too.
//   hist_kernel      one read of the keys -> the 256-bin digit histograms of every radix pass.
//   onesweep_kernel  B3: one LSD pass = one read + one write of keys and values; tiles are handed out
//                    by an atomic ticket, per-digit tile prefixes by decoupled look-back.
//   ranges_kernel    B4: per-tile [start, end) from the sorted keys.
//
// The record count M lives in device memory; every kernel reads it there, so the host needs no
// synchronisation between the stages (grids are sized from capacity_M and surplus blocks exit).
#include "common.cuh"

namespace gs {

// ------------------------------------------------------------------------------ workspace layout
struct BinHeader {
    unsigned long long M;          // total records produced by the emit kernel
    unsigned int emit_ticket;
    unsigned int sort_ticket[8];
    unsigned int pad[5];
};
static_assert(sizeof(BinHeader) == 64, "header size");

constexpr int kRadix = 256;
constexpr int kMaxPasses = 8;

constexpr int kEmitThreads = 256;
constexpr int kEmitItems = 4;
constexpr int kEmitTile = kEmitThreads * kEmitItems;  // entries per block

constexpr int kSortThreads = 256;
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSortItems = 16;
constexpr int kSortTile = kSortThreads * kSortItems;  // keys per block

struct SortPlan {
    int P;
    int shift[kMaxPasses];
    unsigned int mask[kMaxPasses];
};

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Workspace {
    size_t off_header, off_hist, off_emit_status, off_sort_status, zero_bytes, off_keys, off_vals, total;
};
static Workspace layout(int64_t n_entries, int64_t capacity) {
    Workspace w;
    size_t o = 0;
    w.off_header = o; o += sizeof(BinHeader);
    w.off_hist = o; o += (size_t)kMaxPasses * kRadix * sizeof(unsigned int);
    o = align_up(o, 256);
    w.off_emit_status = o; o += (size_t)((n_entries + kEmitTile - 1) / kEmitTile + 1) * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.off_sort_status = o; o += (size_t)((capacity + kSortTile - 1) / kSortTile + 1) * kRadix * sizeof(unsigned long long);
    o = align_up(o, 256);
    w.zero_bytes = o;  // everything up to here is cleared at the start of a call
    w.off_keys = o; o += (size_t)capacity * sizeof(uint64_t);
    o = align_up(o, 256);
    w.off_vals = o; o += (size_t)capacity * sizeof(int32_t);
    o = align_up(o, 256);
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

// ------------------------------------------------------------------------------ B1 + B2
struct EmitArgs {
    int64_t n_entries;      // C * N
    int64_t N;
    int32_t gx, gy;
    int64_t tiles;          // gx * gy
    const float* means2d; const float* depths; const int32_t* radii;
    int64_t capacity;
    uint64_t* keys; int32_t* vals;
    BinHeader* hdr;
    unsigned long long* status;
    int64_t n_blocks;
    unsigned long long* M_dev;
};

__global__ void __launch_bounds__(kEmitThreads) emit_kernel(const EmitArgs a) {
    __shared__ unsigned int s_ticket;
    __shared__ unsigned long long s_base;
    __shared__ unsigned long long s_warp_tiles[kEmitThreads / 32];
    __shared__ unsigned int s_warp_vis[kEmitThreads / 32];
    __shared__ unsigned long long s_off[kEmitTile];   // record offset within the block, compacted
    __shared__ unsigned int s_cnt[kEmitTile];
    __shared__ unsigned int s_xy[kEmitTile];          // x0 | y0 << 16
    __shared__ unsigned int s_w[kEmitTile];
    __shared__ unsigned int s_depth[kEmitTile];
    __shared__ int s_id[kEmitTile];
    __shared__ unsigned int s_nvis;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_ticket = atomicAdd(&a.hdr->emit_ticket, 1u);
    __syncthreads();
    const int64_t tile = s_ticket;
    const int64_t e0 = tile * kEmitTile + (int64_t)tid * kEmitItems;

    int rad[kEmitItems];
    if (e0 + kEmitItems <= a.n_entries) {
        const int4 r4 = __ldg(reinterpret_cast<const int4*>(a.radii + e0));
        rad[0] = r4.x; rad[1] = r4.y; rad[2] = r4.z; rad[3] = r4.w;
    } else {
#pragma unroll
        for (int k = 0; k < kEmitItems; ++k) rad[k] = (e0 + k < a.n_entries) ? __ldg(a.radii + e0 + k) : 0;
    }
    unsigned int cnt[kEmitItems], xy[kEmitItems], ww[kEmitItems], dep[kEmitItems];
    unsigned long long t_tiles = 0;
    unsigned int t_vis = 0;
#pragma unroll
    for (int k = 0; k < kEmitItems; ++k) {
        cnt[k] = 0; xy[k] = 0; ww[k] = 0; dep[k] = 0;
        if (rad[k] > 0) {
            const int64_t e = e0 + k;
            const float2 uv = __ldg(reinterpret_cast<const float2*>(a.means2d) + e);
            int x0, x1, y0, y1;
            tile_rect(uv.x, uv.y, rad[k], a.gx, a.gy, x0, x1, y0, y1);
            ww[k] = (unsigned int)(x1 - x0);
            cnt[k] = ww[k] * (unsigned int)(y1 - y0);
            xy[k] = (unsigned int)x0 | ((unsigned int)y0 << 16);
            if (cnt[k]) {
                dep[k] = __float_as_uint(__ldg(a.depths + e));
                t_tiles += cnt[k];
                ++t_vis;
            }
        }
    }
    // block exclusive scan of (tiles, visible count)
    unsigned long long inc_t = t_tiles;
    unsigned int inc_v = t_vis;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned long long ot = shfl_up_u64(inc_t, d);
        const unsigned int ov = __shfl_up_sync(0xffffffffu, inc_v, d);
        if (lane >= d) { inc_t += ot; inc_v += ov; }
    }
    if (lane == 31) { s_warp_tiles[warp] = inc_t; s_warp_vis[warp] = inc_v; }
    __syncthreads();
    unsigned long long wbase_t = 0, block_tiles = 0;
    unsigned int wbase_v = 0, block_vis = 0;
#pragma unroll
    for (int w = 0; w < kEmitThreads / 32; ++w) {
        if (w < warp) { wbase_t += s_warp_tiles[w]; wbase_v += s_warp_vis[w]; }
        block_tiles += s_warp_tiles[w];
        block_vis += s_warp_vis[w];
    }
    unsigned long long off = wbase_t + inc_t - t_tiles;   // exclusive
    unsigned int ci = wbase_v + inc_v - t_vis;
#pragma unroll
    for (int k = 0; k < kEmitItems; ++k)
        if (cnt[k]) {
            s_off[ci] = off; s_cnt[ci] = cnt[k]; s_xy[ci] = xy[k]; s_w[ci] = ww[k]; s_depth[ci] = dep[k];
            s_id[ci] = (int)(e0 + k);
            off += cnt[k];
            ++ci;
        }
    // decoupled look-back over the preceding blocks' totals (warp 0)
    if (warp == 0) {
        unsigned long long excl = 0;
        if (tile == 0) {
            if (lane == 0) st_volatile_u64(a.status, kFlagIncl | block_tiles);
        } else {
            if (lane == 0) st_volatile_u64(a.status + tile, kFlagAgg | block_tiles);
            int64_t look = tile - 1;
            while (true) {
                const int64_t idx = look - lane;
                unsigned long long st = kFlagIncl;   // virtual predecessor of block 0: inclusive 0
                if (idx >= 0) {
                    do { st = ld_volatile_u64(a.status + idx); } while ((st >> 62) == 0);
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
            if (lane == 0) st_volatile_u64(a.status + tile, kFlagIncl | (excl + block_tiles));
        }
        if (lane == 0) {
            s_base = excl;
            s_nvis = block_vis;
            if (tile == a.n_blocks - 1) {
                a.hdr->M = excl + block_tiles;
                if (a.M_dev) *a.M_dev = excl + block_tiles;
            }
        }
    }
    __syncthreads();
    // warp-cooperative emit: each warp takes visible entries round-robin; its 32 lanes write the
    // entry's records to consecutive addresses
    const unsigned long long base = s_base;
    const unsigned int nvis = s_nvis;
    for (unsigned int j = warp; j < nvis; j += kEmitThreads / 32) {
        const unsigned int c = s_cnt[j], w = s_w[j], xy0 = s_xy[j];
        const unsigned long long o = base + s_off[j];
        const int id = s_id[j];
        const int64_t view = id / a.N;
        const unsigned long long tbase = (unsigned long long)view * (unsigned long long)a.tiles;
        const unsigned int x0 = xy0 & 0xffffu, y0 = xy0 >> 16;
        const unsigned long long lowbits = s_depth[j];
        for (unsigned int k = lane; k < c; k += 32) {
            const unsigned int ry = k / w, rx = k - ry * w;
            const unsigned long long pos = o + k;
            if (pos < (unsigned long long)a.capacity) {
                const unsigned long long t = tbase + (unsigned long long)(y0 + ry) * (unsigned int)a.gx + (x0 + rx);
                a.keys[pos] = (t << 32) | lowbits;
                a.vals[pos] = id;
            }
        }
    }
}

// ------------------------------------------------------------------------------ histograms
__global__ void __launch_bounds__(256) hist_kernel(const uint64_t* __restrict__ keys, const BinHeader* hdr, int64_t capacity,
                                                   const SortPlan plan, unsigned int* __restrict__ hist) {
    __shared__ unsigned int h[kMaxPasses][kRadix];
    for (int k = threadIdx.x; k < kMaxPasses * kRadix; k += blockDim.x) (&h[0][0])[k] = 0;
    __syncthreads();
    const unsigned long long M = hdr->M;
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
    const BinHeader* hdr;
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

    const unsigned long long M = a.hdr->M;
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

// ------------------------------------------------------------------------------ B4
__global__ void __launch_bounds__(256) ranges_kernel(const uint64_t* __restrict__ keys, const BinHeader* hdr, int64_t capacity,
                                                     int64_t* __restrict__ ranges) {
    const unsigned long long M = hdr->M;
    const int64_t n = M < (unsigned long long)capacity ? (int64_t)M : capacity;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t t = (int64_t)(__ldg(keys + i) >> 32);
        if (i == 0) {
            ranges[2 * t] = 0;
        } else {
            const int64_t tp = (int64_t)(__ldg(keys + i - 1) >> 32);
            if (tp != t) {
                ranges[2 * t] = i;
                ranges[2 * tp + 1] = i;
            }
        }
        if (i == n - 1) ranges[2 * t + 1] = n;
    }
}

__global__ void set_count_kernel(BinHeader* hdr, unsigned long long n) { hdr->M = n; }

// run the radix passes; data starts in (k0, v0) and ping-pongs with (k1, v1)
static int run_sort(const SortPlan& plan, uint64_t* k0, int32_t* v0, uint64_t* k1, int32_t* v1, BinHeader* hdr,
                    unsigned int* hist, unsigned long long* status, int64_t capacity, cudaStream_t st) {
    if (plan.P == 0) return GS_OK;
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(onesweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SweepSmem)) != cudaSuccess)
            return GS_ERR_CUDA;
        attr_set = true;
    }
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    hist_kernel<<<sms * 4, 256, 0, st>>>(k0, hdr, capacity, plan, hist);
    int rc = launch_status();
    if (rc) return rc;
    const int64_t tiles = (capacity + kSortTile - 1) / kSortTile;
    for (int p = 0; p < plan.P; ++p) {
        SweepArgs a;
        a.keys_in = (p & 1) ? k1 : k0; a.vals_in = (p & 1) ? v1 : v0;
        a.keys_out = (p & 1) ? k0 : k1; a.vals_out = (p & 1) ? v0 : v1;
        a.hdr = hdr; a.capacity = capacity;
        a.shift = plan.shift[p]; a.mask = plan.mask[p]; a.pass = p;
        a.hist = hist + p * kRadix;
        a.status = status;
        a.ticket = &hdr->sort_ticket[p];
        onesweep_kernel<<<(unsigned)tiles, kSortThreads, sizeof(SweepSmem), st>>>(a);
        rc = launch_status();
        if (rc) return rc;
    }
    return GS_OK;
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
    const int64_t n_entries = (int64_t)C * N;
    const int64_t cap = capacity_M > 0 ? capacity_M : 1;
    const Workspace w = layout(n_entries, cap);
    if (!workspace) {
        if (!workspace_bytes) return GS_ERR_INVALID_ARGUMENT;
        *workspace_bytes = w.total;
        return GS_OK;
    }
    if (workspace_bytes && *workspace_bytes < w.total) return GS_ERR_INVALID_ARGUMENT;
    if (!isect_keys || !isect_vals || !tile_ranges || !aligned(workspace, 256) || !aligned(isect_keys, 8)) return GS_ERR_INVALID_ARGUMENT;
    if (N > 0 && (!means2d || !depths || !radii || !aligned(means2d, 8) || !aligned(radii, 16))) return GS_ERR_INVALID_ARGUMENT;
    cudaStream_t st = (cudaStream_t)stream;
    const int gx = (cams[0].width + kTile - 1) / kTile, gy = (cams[0].height + kTile - 1) / kTile;
    const int64_t tiles = (int64_t)gx * gy;
    int tile_bits = 1;
    while ((1LL << tile_bits) < (int64_t)C * tiles) ++tile_bits;
    const SortPlan plan = make_plan(32 + tile_bits, true);

    unsigned char* ws = reinterpret_cast<unsigned char*>(workspace);
    BinHeader* hdr = reinterpret_cast<BinHeader*>(ws + w.off_header);
    unsigned int* hist = reinterpret_cast<unsigned int*>(ws + w.off_hist);
    unsigned long long* emit_status = reinterpret_cast<unsigned long long*>(ws + w.off_emit_status);
    unsigned long long* sort_status = reinterpret_cast<unsigned long long*>(ws + w.off_sort_status);
    uint64_t* alt_keys = reinterpret_cast<uint64_t*>(ws + w.off_keys);
    int32_t* alt_vals = reinterpret_cast<int32_t*>(ws + w.off_vals);

    if (cudaMemsetAsync(ws, 0, w.zero_bytes, st) != cudaSuccess) return GS_ERR_CUDA;
    if (cudaMemsetAsync(tile_ranges, 0, (size_t)C * tiles * 2 * sizeof(int64_t), st) != cudaSuccess) return GS_ERR_CUDA;
    // with an odd number of passes the records start in the workspace so that they end in the caller's arrays
    uint64_t* k0 = (plan.P & 1) ? alt_keys : isect_keys;
    int32_t* v0 = (plan.P & 1) ? alt_vals : isect_vals;
    uint64_t* k1 = (plan.P & 1) ? isect_keys : alt_keys;
    int32_t* v1 = (plan.P & 1) ? isect_vals : alt_vals;
    const int64_t n_blocks = (n_entries + kEmitTile - 1) / kEmitTile;
    if (n_blocks > 0) {
        EmitArgs a;
        a.n_entries = n_entries; a.N = N; a.gx = gx; a.gy = gy; a.tiles = tiles;
        a.means2d = means2d; a.depths = depths; a.radii = radii;
        a.capacity = capacity_M; a.keys = k0; a.vals = v0;
        a.hdr = hdr; a.status = emit_status; a.n_blocks = n_blocks;
        a.M_dev = reinterpret_cast<unsigned long long*>(M_dev);
        emit_kernel<<<(unsigned)n_blocks, kEmitThreads, 0, st>>>(a);
        rc = launch_status();
        if (rc) return rc;
    } else if (M_dev) {
        if (cudaMemsetAsync(M_dev, 0, sizeof(int64_t), st) != cudaSuccess) return GS_ERR_CUDA;
    }
    if (capacity_M > 0) {
        rc = run_sort(plan, k0, v0, k1, v1, hdr, hist, sort_status, capacity_M, st);
        if (rc) return rc;
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        ranges_kernel<<<sms * 8, 256, 0, st>>>(isect_keys, hdr, capacity_M, tile_ranges);
        rc = launch_status();
        if (rc) return rc;
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

extern "C" int gs_sort_pairs(int64_t n, int32_t end_bit, int32_t skip_bit31, uint64_t* keys, int32_t* vals,
                             void* workspace, size_t* workspace_bytes, void* stream) {
    if (n < 0 || end_bit < 1 || end_bit > 64) return GS_ERR_INVALID_ARGUMENT;
    if (n >= (1LL << 30)) return GS_ERR_UNSUPPORTED;
    const int64_t cap = n > 0 ? n : 1;
    const Workspace w = layout(0, cap);
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
    BinHeader* hdr = reinterpret_cast<BinHeader*>(ws + w.off_header);
    if (cudaMemsetAsync(ws, 0, w.zero_bytes, st) != cudaSuccess) return GS_ERR_CUDA;
    set_count_kernel<<<1, 1, 0, st>>>(hdr, (unsigned long long)n);
    uint64_t* alt_keys = reinterpret_cast<uint64_t*>(ws + w.off_keys);
    int32_t* alt_vals = reinterpret_cast<int32_t*>(ws + w.off_vals);
    int rc = run_sort(plan, keys, vals, alt_keys, alt_vals, hdr, reinterpret_cast<unsigned int*>(ws + w.off_hist),
                      reinterpret_cast<unsigned long long*>(ws + w.off_sort_status), n, st);
    if (rc) return rc;
    if (plan.P & 1) {
        if (cudaMemcpyAsync(keys, alt_keys, (size_t)n * sizeof(uint64_t), cudaMemcpyDeviceToDevice, st) != cudaSuccess) return GS_ERR_CUDA;
        if (cudaMemcpyAsync(vals, alt_vals, (size_t)n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st) != cudaSuccess) return GS_ERR_CUDA;
    }
    return GS_OK;
}
