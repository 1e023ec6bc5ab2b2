// binsort.cu -- xpr_bin_sort: tile binning and the hand-written device radix sort.
//
// Rasterizer stage of the paper: "prefix-sum of tile counts", "replicate",
// "assign tile id" x = x_min + (r mod w), y = y_min + floor(r / w), t = y W' + x, "sort
// lexicographically by (tile id, depth)", "identify bounds".  Key packing tile << 32 | depth bits
// is BASELINE.json:north_star (reading C10); ties keep ascending Gaussian index.
//
// The sort is one stable LSD radix sort of the 64-bit keys, 8 bits per pass, with one observation
// (DESIGN.md section 6): the four low digits are the depth bits, which all pairs of a Gaussian
// share, and replication preserves order.  So the four depth passes run on the visible Gaussians
// (N_vis keys) BEFORE replication, pairs are emitted in that order, and only the tile-id digits
// (2 passes at 1080p) run on the I replicated pairs.  The result is bit-identical to sorting the
// I keys by all digits; HBM traffic per pair drops from 12 + 6*24 + 8 to 12 + 2*24 + 8 bytes.
//
// Kernels (all hand-written, no CUB):
//   compact_kernel   single-pass chained scan (decoupled look-back) of the visibility flags; writes
//                    (depth bits, index) of the visible Gaussians in index order + the 4 depth-digit
//                    histograms.
//   onesweep_kernel  one launch per 8-bit digit, least significant first: warp-striped loads,
//                    stable in-warp ranking (match.any or ballot), shared-memory digit counts,
//                    per-digit decoupled look-back across CTAs, shared-memory staged scatter.
//                    Instantiated for 32-bit keys (Gaussians) and 64-bit keys (pairs).
//   offsets_kernel   chained scan of the tile counts in depth order -> pair offsets and I.
//   emit_kernel      pair-parallel, load-balanced replication (each CTA writes 1024 consecutive pairs:
//                    coalesced 8-byte key / 4-byte value stores) + the tile-digit histograms.
//   ranges_kernel    per-tile (start, end) from the sorted keys.
#include "common.cuh"

namespace xpr {
namespace {

constexpr int RADIX_BITS = 8;
constexpr int RADIX = 1 << RADIX_BITS;
constexpr int DEPTH_PASSES = 4;             // 32 depth bits
constexpr int MAX_TILE_PASSES = 4;          // up to 2^31 tiles

constexpr int SCAN_THREADS = 256;           // Gaussians per compact / emit block (one per thread)
constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
static_assert(SORT_THREADS == RADIX, "one thread per digit");
constexpr int IPT32 = 4;                    // Gaussian-level passes: 1024 keys per CTA (N_vis is small)
constexpr int IPT64 = 16;                   // pair-level passes: 4096 pairs per CTA

constexpr uint32_t FLAG_PARTIAL = 1u << 30, FLAG_INCLUSIVE = 2u << 30, FLAG_MASK = 3u << 30, VALUE_MASK = ~FLAG_MASK;
constexpr unsigned long long SFLAG_PARTIAL = 1ull << 62, SFLAG_INCLUSIVE = 2ull << 62, SFLAG_MASK = 3ull << 62;

// Header at the start of the workspace (zeroed every call).
struct Header {
    unsigned long long total_pairs;          // I
    uint32_t n_vis;                          // visible Gaussians
    uint32_t compact_ticket, emit_ticket;
    uint32_t sort_ticket[DEPTH_PASSES + MAX_TILE_PASSES];
    uint32_t pad[5];
    uint32_t hist[(DEPTH_PASSES + MAX_TILE_PASSES) * RADIX];   // global digit histograms
};

struct Layout {
    size_t header, scan_status, vkey0, vidx0, vkey1, vidx1, status32, keys_tmp, vals_tmp, status64, total;
};

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

inline int tile_passes_for(int32_t num_tiles) {
    int bits = 0;
    while (bits < 31 && ((int64_t)1 << bits) < (int64_t)num_tiles) ++bits;
    return (bits + RADIX_BITS - 1) / RADIX_BITS;
}

inline Layout make_layout(int64_t N, int64_t cap, int32_t num_tiles) {
    Layout L;
    size_t off = 0;
    const size_t n = (size_t)N, c = (size_t)cap;
    const size_t scan_blocks = (n + SCAN_THREADS - 1) / SCAN_THREADS;
    L.header = off; off = align_up(off + sizeof(Header), 256);
    L.scan_status = off; off = align_up(off + 8 * 2 * (scan_blocks + 1), 256);      // compact + emit chains
    const size_t tiles32 = (n + SORT_THREADS * IPT32 - 1) / (SORT_THREADS * IPT32);
    L.status32 = off; off = align_up(off + 4 * (size_t)RADIX * tiles32 * DEPTH_PASSES, 256);
    // everything up to here is zeroed with one memset
    L.vkey0 = off; off = align_up(off + 4 * n, 256);
    L.vidx0 = off; off = align_up(off + 4 * n, 256);
    L.vkey1 = off; off = align_up(off + 4 * n, 256);
    L.vidx1 = off; off = align_up(off + 4 * n, 256);
    L.keys_tmp = off; off = align_up(off + 8 * c, 256);
    L.vals_tmp = off; off = align_up(off + 4 * c, 256);
    const size_t tiles64 = (c + SORT_THREADS * IPT64 - 1) / (SORT_THREADS * IPT64);
    L.status64 = off; off = align_up(off + 4 * (size_t)RADIX * tiles64 * (size_t)tile_passes_for(num_tiles), 256);
    L.total = off;
    return L;
}

__device__ __forceinline__ uint32_t ld_relaxed(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed(uint32_t* p, uint32_t v) {
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_relaxed64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Block-wide exclusive scan of one value per thread (SCAN_THREADS threads) followed by the chained
// scan across blocks (decoupled look-back; `block` is a ticket, so predecessors are running or done).
// Returns the block-local exclusive offset; *block_total and *global_base are block-uniform.
__device__ __forceinline__ uint32_t chained_scan(uint32_t x, uint32_t block, unsigned long long* __restrict__ status,
                                                 uint32_t* s_warp, unsigned long long* s_base, uint32_t* block_total,
                                                 unsigned long long* global_base) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint32_t wbase = 0, btotal = 0;
#pragma unroll
    for (int w = 0; w < SCAN_THREADS / 32; ++w) {
        const uint32_t v = s_warp[w];
        if (w < warp) wbase += v;
        btotal += v;
    }
    if (warp == 0) {
        // decoupled look-back by one warp: 32 predecessors per step
        unsigned long long excl = 0;
        if (block == 0) {
            if (lane == 0) st_relaxed64(&status[0], SFLAG_INCLUSIVE | (unsigned long long)btotal);
        } else {
            if (lane == 0) st_relaxed64(&status[block], SFLAG_PARTIAL | (unsigned long long)btotal);
            int64_t top = (int64_t)block - 1;          // lane l inspects predecessor top - l
            while (true) {
                const int64_t t = top - lane;
                unsigned long long sv = SFLAG_INCLUSIVE;   // virtual predecessors before block 0: inclusive 0
                if (t >= 0) { do { sv = ld_relaxed64(&status[t]); } while ((sv & SFLAG_MASK) == 0); }
                const uint32_t incl_mask = __ballot_sync(0xffffffffu, (sv & SFLAG_MASK) == SFLAG_INCLUSIVE);
                const int first = incl_mask ? (__ffs(incl_mask) - 1) : 32;     // nearest inclusive predecessor
                unsigned long long v = (lane <= first) ? (sv & ~SFLAG_MASK) : 0ull;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                excl += v;
                if (incl_mask) break;
                top -= 32;
            }
            if (lane == 0) st_relaxed64(&status[block], SFLAG_INCLUSIVE | (excl + btotal));
        }
        if (lane == 0) *s_base = excl;
    }
    __syncthreads();
    *block_total = btotal;
    *global_base = *s_base;
    return wbase + incl - x;
}

// ---------------------------------------------------------------------------------------------
// compact: visible Gaussians in index order -> (depth bits, index), + depth-digit histograms
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SCAN_THREADS)
compact_kernel(int64_t N, const float* __restrict__ depth, const uint32_t* __restrict__ tcount,
               Header* __restrict__ hdr, unsigned long long* __restrict__ status, uint32_t* __restrict__ vkey,
               uint32_t* __restrict__ vidx) {
    __shared__ uint32_t s_warp[SCAN_THREADS / 32];
    __shared__ uint32_t s_hist[DEPTH_PASSES * RADIX];
    __shared__ uint32_t s_block;
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x;
    if (tid == 0) s_block = atomicAdd(&hdr->compact_ticket, 1u);
    for (int b = tid; b < DEPTH_PASSES * RADIX; b += SCAN_THREADS) s_hist[b] = 0u;
    __syncthreads();
    const uint32_t block = s_block;
    const int64_t i = (int64_t)block * SCAN_THREADS + tid;
    const bool vis = (i < N) && (tcount[i] != 0u);
    uint32_t db = 0;
    if (vis) {
        db = __float_as_uint(depth[i]);
#pragma unroll
        for (int d = 0; d < DEPTH_PASSES; ++d) atomicAdd(&s_hist[d * RADIX + ((db >> (8 * d)) & 255u)], 1u);
    }
    uint32_t btotal; unsigned long long base;
    const uint32_t off = chained_scan(vis ? 1u : 0u, block, status, s_warp, &s_base, &btotal, &base);
    if (vis) {
        vkey[base + off] = db;
        vidx[base + off] = (uint32_t)i;
    }
    if (tid == 0 && (int64_t)(block + 1) * SCAN_THREADS >= N) hdr->n_vis = (uint32_t)(base + btotal);
    for (int b = tid; b < DEPTH_PASSES * RADIX; b += SCAN_THREADS) {
        const uint32_t v = s_hist[b];
        if (v) atomicAdd(&hdr->hist[b], v);
    }
}

// ---------------------------------------------------------------------------------------------
// offsets: chained scan of the tile counts in depth order ("prefix-sum of tile counts")
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SCAN_THREADS)
offsets_kernel(const uint32_t* __restrict__ vidx, const uint32_t* __restrict__ tcount, Header* __restrict__ hdr,
               unsigned long long* __restrict__ status, uint32_t* __restrict__ voff) {
    __shared__ uint32_t s_warp[SCAN_THREADS / 32];
    __shared__ uint32_t s_block;
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x;
    const uint32_t n_vis = hdr->n_vis;
    if (tid == 0) s_block = atomicAdd(&hdr->emit_ticket, 1u);   // ticket order = look-back order
    __syncthreads();
    const uint32_t block = s_block;
    if ((uint64_t)block * SCAN_THREADS >= n_vis && block != 0) return;   // beyond the visible list: nobody waits on us
    const uint32_t s = block * SCAN_THREADS + tid;       // position in depth order
    const uint32_t tc = (s < n_vis) ? tcount[vidx[s]] : 0u;
    uint32_t btotal; unsigned long long base;
    const uint32_t off = chained_scan(tc, block, status, s_warp, &s_base, &btotal, &base);
    if (s < n_vis) voff[s] = (uint32_t)(base + off);     // only used when I <= pair_capacity < 2^30
    if (tid == 0 && (uint64_t)(block + 1) * SCAN_THREADS >= n_vis) hdr->total_pairs = base + btotal;   // I
}

// ---------------------------------------------------------------------------------------------
// emit: replicate + assign tile id, pair-parallel and load-balanced: CTA b writes the
// pairs [b*EMIT_PAIRS, (b+1)*EMIT_PAIRS) whatever Gaussians they belong to (a near Gaussian may
// cover thousands of tiles, and in depth order those come first).  + tile-digit histograms.
// ---------------------------------------------------------------------------------------------
constexpr int EMIT_THREADS = 256, EMIT_PPT = 4, EMIT_PAIRS = EMIT_THREADS * EMIT_PPT;

__global__ void __launch_bounds__(EMIT_THREADS)
emit_kernel(uint32_t I, int TW, int tile_passes, const uint32_t* __restrict__ vkey, const uint32_t* __restrict__ vidx,
            const uint32_t* __restrict__ voff, const int4* __restrict__ rect, Header* __restrict__ hdr,
            uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
    __shared__ uint32_t s_off[EMIT_PAIRS + 1];       // pair offsets of the Gaussians this CTA touches
    __shared__ int s_x0[EMIT_PAIRS], s_y0[EMIT_PAIRS], s_w[EMIT_PAIRS];
    __shared__ uint32_t s_dbits[EMIT_PAIRS], s_gid[EMIT_PAIRS];
    __shared__ uint32_t s_hist[MAX_TILE_PASSES * RADIX];
    __shared__ uint32_t s_first;
    const int tid = threadIdx.x, lane = tid & 31;
    const uint32_t n_vis = hdr->n_vis;
    const uint32_t p0 = blockIdx.x * (uint32_t)EMIT_PAIRS, p1 = min(I, p0 + (uint32_t)EMIT_PAIRS);
    for (int b = tid; b < tile_passes * RADIX; b += EMIT_THREADS) s_hist[b] = 0u;
    if (tid == 0) {      // last Gaussian (in depth order) whose offset is <= p0
        uint32_t lo = 0, hi = n_vis;                 // invariant: voff[lo] <= p0, (hi == n_vis or voff[hi] > p0)
        while (hi - lo > 1) {
            const uint32_t mid = (lo + hi) >> 1;
            if (voff[mid] <= p0) lo = mid; else hi = mid;
        }
        s_first = lo;
    }
    __syncthreads();
    const uint32_t first = s_first;
    // Gaussians first .. first+cnt-1 cover [p0, p1); cnt <= EMIT_PAIRS because every listed Gaussian
    // after the first starts inside the range
    uint32_t cnt = 0;
    for (uint32_t k = tid; k < (uint32_t)EMIT_PAIRS; k += EMIT_THREADS) {
        const uint32_t s = first + k;
        uint32_t off = 0xffffffffu;
        if (s < n_vis) off = voff[s];
        if (s < n_vis && off < p1) {
            const uint32_t g = vidx[s];
            const int4 r = rect[g];
            s_off[k] = off; s_x0[k] = r.x; s_y0[k] = r.y; s_w[k] = r.z - r.x; s_dbits[k] = vkey[s]; s_gid[k] = g;
        } else {
            s_off[k] = 0xffffffffu;                  // sentinel: never <= a pair index
        }
    }
    if (tid == 0) s_off[EMIT_PAIRS] = 0xffffffffu;
    __syncthreads();
    (void)cnt;
#pragma unroll
    for (int it = 0; it < EMIT_PPT; ++it) {
        const uint32_t j = p0 + (uint32_t)it * EMIT_THREADS + tid;
        const bool valid = j < p1;
        uint32_t tile = 0;
        if (valid) {
            int lo = 0, hi = EMIT_PAIRS;             // invariant: s_off[lo] <= j < s_off[hi]
#pragma unroll
            for (int q = 0; q < 10; ++q) {
                const int mid = (lo + hi) >> 1;
                if (s_off[mid] <= j) lo = mid; else hi = mid;
            }
            const uint32_t r = j - s_off[lo];
            const uint32_t w = (uint32_t)s_w[lo];
            const uint32_t ry = r / w, rx = r - ry * w;
            tile = (uint32_t)(s_y0[lo] + (int)ry) * (uint32_t)TW + (uint32_t)(s_x0[lo] + (int)rx);
            keys[j] = ((uint64_t)tile << 32) | (uint64_t)s_dbits[lo];
            vals[j] = s_gid[lo];
            if (tile_passes > 0) atomicAdd(&s_hist[tile & 255u], 1u);   // consecutive tiles -> distinct banks
        }
        // higher tile digits are nearly warp-uniform: aggregate with match.any before the atomic
        for (int d = 1; d < tile_passes; ++d) {
            const uint32_t dig = valid ? ((tile >> (8 * d)) & 255u) : 0xffffffffu;
            const uint32_t peers = __match_any_sync(0xffffffffu, dig);
            if (valid && (peers & ((1u << lane) - 1u)) == 0u) atomicAdd(&s_hist[d * RADIX + dig], (uint32_t)__popc(peers));
        }
    }
    __syncthreads();
    for (int b = tid; b < tile_passes * RADIX; b += EMIT_THREADS) {
        const uint32_t v = s_hist[b];
        if (v) atomicAdd(&hdr->hist[DEPTH_PASSES * RADIX + b], v);
    }
}

// ---------------------------------------------------------------------------------------------
// onesweep digit pass (KeyT = uint32_t for Gaussians, uint64_t for pairs)
// ---------------------------------------------------------------------------------------------
template <class KeyT, int IPT>
struct SortSmem {
    KeyT keys[SORT_THREADS * IPT];
    uint32_t vals[SORT_THREADS * IPT];
    uint32_t warp_hist[SORT_WARPS][RADIX];
    uint32_t cta_excl[RADIX];     // exclusive digit offsets inside the tile
    uint32_t gbase[RADIX];        // global position of digit d's first key of this tile, minus cta_excl[d]
    uint32_t scan_tmp[SORT_WARPS];
    uint32_t tile_id;
};

// BALLOT = true: peer mask from 8 ballots (cost independent of the digit distribution);
// false: match.any (fast when a warp holds few distinct digits, slow when it holds 32).
template <class KeyT, int IPT, bool BALLOT>
__global__ void __launch_bounds__(SORT_THREADS)
onesweep_kernel(const uint32_t* __restrict__ n_dev32, const unsigned long long* __restrict__ n_dev64, int shift,
                int hist_row, int ticket_row, const KeyT* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                KeyT* __restrict__ keys_out, uint32_t* __restrict__ vals_out, Header* __restrict__ hdr,
                uint32_t* __restrict__ status /* [tiles][RADIX] of this pass */) {
    constexpr int TILE_KEYS = SORT_THREADS * IPT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem<KeyT, IPT>& S = *reinterpret_cast<SortSmem<KeyT, IPT>*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t n = n_dev32 ? *n_dev32 : (uint32_t)*n_dev64;

    if (tid == 0) S.tile_id = atomicAdd(&hdr->sort_ticket[ticket_row], 1u);
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) S.warp_hist[w][tid] = 0u;    // SORT_THREADS == RADIX
    __syncthreads();
    const uint32_t tile = S.tile_id;
    if ((uint64_t)tile * TILE_KEYS >= n) return;                      // grid is sized for an upper bound of n
    const uint32_t tile_base = tile * (uint32_t)TILE_KEYS;
    const uint32_t tile_n = min((uint32_t)TILE_KEYS, n - tile_base);

    // warp-striped load: item `it` of lane l of warp w sits at tile_base + w*32*IPT + it*32 + l
    KeyT key[IPT];
    uint32_t val[IPT];
    const uint32_t wofs = (uint32_t)warp * 32u * IPT + (uint32_t)lane;
#pragma unroll
    for (int it = 0; it < IPT; ++it) {
        const uint32_t loc = wofs + (uint32_t)it * 32u;
        if (loc < tile_n) {
            key[it] = keys_in[tile_base + loc];
            val[it] = vals_in[tile_base + loc];
        } else {
            key[it] = ~(KeyT)0;    // padding: highest digit, ranks after every real key of the tile
            val[it] = 0u;
        }
    }
    // stable in-warp ranking: rank = #earlier items of this warp with the same digit
    uint32_t rank[IPT];
    const uint32_t lt_mask = (1u << lane) - 1u;
#pragma unroll
    for (int it = 0; it < IPT; ++it) {
        const uint32_t d = (uint32_t)(key[it] >> shift) & (RADIX - 1);
        uint32_t peers;
        if (BALLOT) {
            peers = 0xffffffffu;
#pragma unroll
            for (int b = 0; b < RADIX_BITS; ++b) {
                const bool bit = (d >> b) & 1u;
                const uint32_t m = __ballot_sync(0xffffffffu, bit);
                peers &= bit ? m : ~m;
            }
        } else {
            peers = __match_any_sync(0xffffffffu, d);
        }
        const uint32_t lt = peers & lt_mask;
        uint32_t prev = 0;
        if (lt == 0u) {                                  // lowest lane of the peer group
            prev = S.warp_hist[warp][d];
            S.warp_hist[warp][d] = prev + (uint32_t)__popc(peers);
        }
        __syncwarp();
        prev = __shfl_sync(0xffffffffu, prev, __ffs(peers) - 1);
        rank[it] = prev + (uint32_t)__popc(lt);
    }
    __syncthreads();
    // per digit (thread tid == digit): exclusive scan over warps, CTA count
    uint32_t count = 0;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) {
        const uint32_t v = S.warp_hist[w][tid];
        S.warp_hist[w][tid] = count;
        count += v;
    }
    // the last tile's padding was counted in digit RADIX-1: remove it from what look-back publishes
    uint32_t real_count = count;
    if (tid == RADIX - 1) real_count -= (uint32_t)TILE_KEYS - tile_n;
    // block exclusive scan over digits of `count` -> cta_excl; and of the global histogram -> bin base
    const uint32_t gh = hdr->hist[hist_row * RADIX + tid];
    uint32_t inc_c = count, inc_g = gh;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t a = __shfl_up_sync(0xffffffffu, inc_c, o), b = __shfl_up_sync(0xffffffffu, inc_g, o);
        if (lane >= o) { inc_c += a; inc_g += b; }
    }
    if (lane == 31) { S.scan_tmp[warp] = inc_c; S.cta_excl[warp] = inc_g; }   // cta_excl reused as scratch
    __syncthreads();
    uint32_t pre_c = 0, pre_g = 0;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w)
        if (w < warp) { pre_c += S.scan_tmp[w]; pre_g += S.cta_excl[w]; }
    __syncthreads();
    const uint32_t excl_c = pre_c + inc_c - count;        // position of digit tid inside the tile
    const uint32_t bin_base = pre_g + inc_g - gh;         // global position of digit tid's first key
    S.cta_excl[tid] = excl_c;
    // decoupled look-back over earlier tiles, one thread per digit
    uint32_t* my = status + (size_t)tile * RADIX + tid;
    uint32_t excl_prev = 0;
    if (tile == 0) {
        st_relaxed(my, FLAG_INCLUSIVE | real_count);
    } else {
        st_relaxed(my, FLAG_PARTIAL | real_count);
        const uint32_t* p = my - RADIX;
        uint32_t remaining = tile;
        bool found = false;
        while (!found) {   // 4 predecessors in flight per round; before tile 0: virtual inclusive 0
            uint32_t sv[4];
#pragma unroll
            for (int k = 0; k < 4; ++k)
                sv[k] = ((uint32_t)k < remaining) ? ld_relaxed(p - k * RADIX) : FLAG_INCLUSIVE;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (found) break;
                while ((sv[k] & FLAG_MASK) == 0u) sv[k] = ld_relaxed(p - k * RADIX);
                excl_prev += sv[k] & VALUE_MASK;
                found = (sv[k] & FLAG_MASK) == FLAG_INCLUSIVE;
            }
            p -= 4 * RADIX;
            remaining = (remaining > 4u) ? remaining - 4u : 0u;
        }
        st_relaxed(my, FLAG_INCLUSIVE | (excl_prev + real_count));
    }
    S.gbase[tid] = bin_base + excl_prev - excl_c;
    __syncthreads();
    // scatter into shared memory in tile-sorted order
#pragma unroll
    for (int it = 0; it < IPT; ++it) {
        const uint32_t d = (uint32_t)(key[it] >> shift) & (RADIX - 1);
        const uint32_t pos = S.cta_excl[d] + S.warp_hist[warp][d] + rank[it];
        S.keys[pos] = key[it];
        S.vals[pos] = val[it];
    }
    __syncthreads();
    // coalesced runs to global memory (padding sits at positions >= tile_n)
#pragma unroll
    for (int it = 0; it < IPT; ++it) {
        const uint32_t p = (uint32_t)it * SORT_THREADS + (uint32_t)tid;
        if (p < tile_n) {
            const KeyT k = S.keys[p];
            const uint32_t d = (uint32_t)(k >> shift) & (RADIX - 1);
            const uint32_t dst = S.gbase[d] + p;
            keys_out[dst] = k;
            vals_out[dst] = S.vals[p];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// per-tile bounds ("records each segment's start b_j and count c_j")
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
ranges_kernel(uint32_t I, const uint64_t* __restrict__ keys, uint32_t* __restrict__ ranges) {
    const uint32_t j = blockIdx.x * 256u + threadIdx.x;
    if (j >= I) return;
    const uint32_t t = (uint32_t)(keys[j] >> 32);
    if (j == 0 || (uint32_t)(keys[j - 1] >> 32) != t) ranges[2 * t] = j;
    if (j == I - 1 || (uint32_t)(keys[j + 1] >> 32) != t) ranges[2 * t + 1] = j + 1;
}

}  // namespace
}  // namespace xpr

using namespace xpr;

extern "C" int32_t xpr_bin_sort_workspace(int64_t N, int64_t pair_capacity, int32_t num_tiles, size_t* bytes) {
    if (!bytes || N < 0 || N > 0x7fffffffLL || pair_capacity < 0 || pair_capacity >= (1LL << 30) || num_tiles <= 0)
        return XPR_ERR_INVALID_ARG;
    *bytes = make_layout(N, pair_capacity, num_tiles).total;
    return XPR_OK;
}

template <class KeyT, int IPT, bool BALLOT>
static cudaError_t launch_pass(unsigned grid, cudaStream_t st, const uint32_t* n32, const unsigned long long* n64,
                               int shift, int row, const KeyT* kin, const uint32_t* vin, KeyT* kout, uint32_t* vout,
                               Header* hdr, uint32_t* status) {
    const size_t smem = sizeof(SortSmem<KeyT, IPT>);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(onesweep_kernel<KeyT, IPT, BALLOT>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    onesweep_kernel<KeyT, IPT, BALLOT><<<grid, SORT_THREADS, smem, st>>>(n32, n64, shift, row, row, kin, vin, kout,
                                                                        vout, hdr, status);
    return cudaGetLastError();
}

extern "C" int32_t xpr_bin_sort(int64_t N, const float* depth, const int32_t* tile_rect, const uint32_t* tile_count,
                                const xpr_camera* cam, const xpr_config* cfg, int64_t pair_capacity,
                                uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* tile_ranges,
                                int64_t* num_pairs_host, void* workspace, size_t workspace_bytes, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0 || N > 0x7fffffffLL || pair_capacity < 0 || pair_capacity >= (1LL << 30) || !num_pairs_host)
        return XPR_ERR_INVALID_ARG;
    const int TW = tiles_x(cam), TH = tiles_y(cam);
    const int64_t T64 = (int64_t)TW * TH;
    if (T64 > 0x7fffffffLL) return XPR_ERR_UNSUPPORTED;
    const int32_t T = (int32_t)T64;
    if (!aligned(tile_ranges, 8) || !aligned(workspace, 256)) return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(depth, 4) || !aligned(tile_rect, 16) || !aligned(tile_count, 4))) return XPR_ERR_INVALID_ARG;
    if (pair_capacity > 0 && (!aligned(keys_sorted, 8) || !aligned(vals_sorted, 4))) return XPR_ERR_INVALID_ARG;
    const Layout L = make_layout(N, pair_capacity, T);
    if (workspace_bytes < L.total) return XPR_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    Header* hdr = reinterpret_cast<Header*>(ws + L.header);
    const size_t scan_blocks = ((size_t)N + SCAN_THREADS - 1) / SCAN_THREADS;
    unsigned long long* compact_status = reinterpret_cast<unsigned long long*>(ws + L.scan_status);
    unsigned long long* emit_status = compact_status + scan_blocks + 1;
    uint32_t* vkey[2] = {reinterpret_cast<uint32_t*>(ws + L.vkey0), reinterpret_cast<uint32_t*>(ws + L.vkey1)};
    uint32_t* vidx[2] = {reinterpret_cast<uint32_t*>(ws + L.vidx0), reinterpret_cast<uint32_t*>(ws + L.vidx1)};
    uint32_t* status32 = reinterpret_cast<uint32_t*>(ws + L.status32);
    uint64_t* keys_tmp = reinterpret_cast<uint64_t*>(ws + L.keys_tmp);
    uint32_t* vals_tmp = reinterpret_cast<uint32_t*>(ws + L.vals_tmp);
    uint32_t* status64 = reinterpret_cast<uint32_t*>(ws + L.status64);
    const int tpasses = tile_passes_for(T);

    XPR_CUDA(cudaMemsetAsync(tile_ranges, 0, sizeof(uint32_t) * 2 * (size_t)T, st));
    *num_pairs_host = 0;
    if (N == 0) return XPR_OK;
    XPR_CUDA(cudaMemsetAsync(ws + L.header, 0, L.vkey0 - L.header, st));   // header, scan chains, status32
    // 1. visible Gaussians (index order) + depth-digit histograms
    compact_kernel<<<(unsigned)scan_blocks, SCAN_THREADS, 0, st>>>(N, depth, tile_count, hdr, compact_status, vkey[0],
                                                                   vidx[0]);
    XPR_LAUNCH_CHECK();
    // 2. the four depth digits, on the N_vis Gaussians (grid sized for N; surplus CTAs exit)
    const unsigned tiles32 = (unsigned)(((size_t)N + SORT_THREADS * IPT32 - 1) / (SORT_THREADS * IPT32));
    for (int p = 0; p < DEPTH_PASSES; ++p) {
        uint32_t* status = status32 + (size_t)p * RADIX * tiles32;
        const int a = p & 1, b = a ^ 1;
        cudaError_t e = (p < 3)   // mantissa bytes: ~32 distinct digits per warp -> ballot ranking
            ? launch_pass<uint32_t, IPT32, true>(tiles32, st, &hdr->n_vis, nullptr, 8 * p, p, vkey[a], vidx[a], vkey[b], vidx[b], hdr, status)
            : launch_pass<uint32_t, IPT32, false>(tiles32, st, &hdr->n_vis, nullptr, 8 * p, p, vkey[a], vidx[a], vkey[b], vidx[b], hdr, status);
        XPR_CUDA(e);
    }   // DEPTH_PASSES is even: the sorted list is back in vkey[0] / vidx[0]
    // 3. pair offsets in depth order and the pair count I (the one host read-back)
    uint32_t* voff = vkey[1];                          // free after the depth passes
    offsets_kernel<<<(unsigned)scan_blocks, SCAN_THREADS, 0, st>>>(vidx[0], tile_count, hdr, emit_status, voff);
    XPR_LAUNCH_CHECK();
    unsigned long long total = 0;
    XPR_CUDA(cudaMemcpyAsync(&total, &hdr->total_pairs, sizeof(total), cudaMemcpyDeviceToHost, st));
    XPR_CUDA(cudaStreamSynchronize(st));
    *num_pairs_host = (int64_t)total;
    if ((int64_t)total > pair_capacity) return XPR_ERR_CAPACITY;
    if (total == 0) return XPR_OK;
    const uint32_t I = (uint32_t)total;
    // replicate in depth order; an even number of tile passes ends in the buffer emission wrote to
    uint64_t* k0 = (tpasses % 2 == 0) ? keys_sorted : keys_tmp;
    uint32_t* v0 = (tpasses % 2 == 0) ? vals_sorted : vals_tmp;
    uint64_t* k1 = (tpasses % 2 == 0) ? keys_tmp : keys_sorted;
    uint32_t* v1 = (tpasses % 2 == 0) ? vals_tmp : vals_sorted;
    emit_kernel<<<(I + EMIT_PAIRS - 1) / EMIT_PAIRS, EMIT_THREADS, 0, st>>>(
        I, TW, tpasses, vkey[0], vidx[0], voff, reinterpret_cast<const int4*>(tile_rect), hdr, k0, v0);
    XPR_LAUNCH_CHECK();
    // 4. the tile-id digits, on the I pairs
    const unsigned tiles64 = (I + SORT_THREADS * IPT64 - 1) / (SORT_THREADS * IPT64);
    if (tpasses > 0) XPR_CUDA(cudaMemsetAsync(status64, 0, sizeof(uint32_t) * (size_t)RADIX * tiles64 * (size_t)tpasses, st));
    for (int p = 0; p < tpasses; ++p) {
        uint32_t* status = status64 + (size_t)p * RADIX * tiles64;
        const int row = DEPTH_PASSES + p;
        cudaError_t e = (p == 0)  // consecutive pairs of a Gaussian are consecutive tiles -> ballot ranking
            ? launch_pass<uint64_t, IPT64, true>(tiles64, st, nullptr, &hdr->total_pairs, 32 + 8 * p, row, k0, v0, k1, v1, hdr, status)
            : launch_pass<uint64_t, IPT64, false>(tiles64, st, nullptr, &hdr->total_pairs, 32 + 8 * p, row, k0, v0, k1, v1, hdr, status);
        XPR_CUDA(e);
        uint64_t* tk = k0; k0 = k1; k1 = tk;
        uint32_t* tv = v0; v0 = v1; v1 = tv;
    }
    ranges_kernel<<<(I + 255) / 256, 256, 0, st>>>(I, keys_sorted, tile_ranges);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}
