// binsort.cu -- xpr_bin_sort / xpr_bin_sort_cull: tile binning and the hand-written device radix sort.
//
// Rasterizer stage of the paper: "prefix-sum of tile counts", "replicate",
// "assign tile id" x = x_min + (r mod w), y = y_min + floor(r / w), t = y W' + x, optional "cull"
// (tile_cull, Listing 1), "sort lexicographically by (tile id, depth)", "identify bounds".
// Key packing tile << 32 | depth bits is BASELINE.json:north_star (reading C10); ties keep ascending
// Gaussian index.
//
// The result is the stable LSD radix sort of the I (key, value) pairs by all 32 + log2(T) key bits --
// bit-identical, checked against std::stable_sort -- but the pairs themselves are written exactly once,
// at their final position:
//  (1) the four low digits are the depth bits, which all pairs of a Gaussian share.  The four depth
//      passes therefore run on the visible Gaussians (N_vis keys, not I), giving every Gaussian its
//      RANK in (depth, index) order.
//  (2) a ROW is the run of consecutive tiles one Gaussian covers in one tile row: tile_cull reduces to
//      one surviving interval per row (the quadratic form is convex), found with 3-4 evaluations of the
//      exact per-tile predicate instead of one per tile; pairs that fail tile_cull never exist.  A row is
//      stored as (first column, length) and also adds +1 / -1 to a difference array over the tile ids,
//      whose two prefix sums are the per-tile counts and the per-tile bases ("identify bounds", without
//      looking at a single pair).
//  (3) the tile digits are sorted MOST significant first, on a coarse level: a SUPERTILE is a block of
//      8 x 8 tiles; a Gaussian emits one 8-byte word (supertile << 32 | rank) per supertile its rectangle
//      touches (~2 per Gaussian instead of ~33 pairs), and ONE stable onesweep pass per 8 bits of the
//      supertile id sorts those words: afterwards every supertile owns a segment of Gaussians in rank order.
//  (4) the final pass walks a segment in chunks of 256 words.  A word expands to the 64-bit mask of the
//      tiles its Gaussian covers inside the supertile (from the row table); the position of a pair inside
//      its tile is the number of earlier Gaussians of the segment whose mask has the same bit -- a ballot
//      and a popcount per (warp, tile), a per-(chunk, tile) count, and a decoupled look-back over the
//      earlier chunks of the segment.  Every thread then writes key = tile << 32 | depth bits and value =
//      Gaussian index of its pairs at tile base + position.
// HBM traffic per pair: 12 bytes written once (8 + 4), against 12 + 6 * 24 + 8 = 164 bytes for the plain
// six-pass key-value sort and 44 bytes for sorting packed pair words in two tile passes.  No count ever
// travels to the host inside the call (persistent grids; optional read-back at the end).
//
// Kernels (all hand-written, no CUB):
//   compact_kernel    single-pass chained scan (decoupled look-back) of the visibility flags; writes
//                     (depth bits, index) of the visible Gaussians in index order + the 4 depth-digit
//                     histograms.
//   onesweep_kernel   one launch per 8-bit digit, least significant first: warp-striped loads, stable
//                     in-warp ranking (shared-memory bitmap or match.any), shared-memory digit counts,
//                     per-digit decoupled look-back across tiles, shared-memory staged scatter.
//                     Instantiated for 32-bit keys + values (depth passes on the Gaussians) and for
//                     64-bit words (the supertile pass).
//   rank_scan_kernel  chained scan, in rank order, of the rows and of the supertiles of every Gaussian.
//   rows_kernel       one thread per row: surviving interval (tile_cull) -> row table + difference array.
//   l1_emit_kernel    one thread per Gaussian: its supertile words, the supertile digit histograms and
//                     the per-supertile counts.
//   tile_scan_kernel  one CTA: per-tile counts and bases -> tile_ranges, I, the capacity verdict; the
//                     segment and chunk tables of the supertiles.
//   final_kernel      per chunk of a supertile segment: masks, ballot ranking, look-back, scatter.
#include "common.cuh"
#include <mutex>

namespace xpr {
namespace {

// Programmatic dependent launch (sm_90+) between the kernels of one xpr_bin_sort call.  A kernel launched with the
// attribute may be scheduled as soon as every CTA of its predecessor has issued griddepcontrol.launch_dependents (all
// kernels here do so first thing), and must execute griddepcontrol.wait -- which returns once the predecessor grid has
// COMPLETED and its writes are visible -- before it touches anything.  The dependency is unchanged; launch latency and
// CTA scheduling of kernel k+1 overlap the tail of kernel k.  Measured per launch site (config 3 / config 5, bin_sort
// stage): off 0.182 / 0.804 ms; on everywhere 0.177 / 0.875 ms (the early l1_emit CTAs take SM slots from the
// long-running rows kernel); on everywhere except l1_emit 0.166 / 0.793 ms -- kept.
#ifndef XPR_PDL
#define XPR_PDL 1
#endif
__device__ __forceinline__ void pdl_entry() {
#if XPR_PDL
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
}
template <class... KArgs, class... Args>
static cudaError_t launch_k(bool pdl, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                            Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = (XPR_PDL && pdl) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

constexpr int RADIX_BITS = 8;
constexpr int RADIX = 1 << RADIX_BITS;
constexpr int DEPTH_PASSES = 4;             // 32 depth bits
constexpr int MAX_TILE_PASSES = 4;          // up to 2^31 supertiles

constexpr int SCAN_THREADS = 256;           // compact / rank scan: 8 warps x 256 items
constexpr int SCAN_WARPS = SCAN_THREADS / 32;
constexpr int SCAN_ROUNDS = 8;              // items per lane
constexpr int SCAN_ITEMS = SCAN_THREADS * SCAN_ROUNDS;
constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
static_assert(SORT_THREADS == RADIX, "one thread per digit");
constexpr int IPT32 = 4;                    // Gaussian-level passes: 1024 keys per tile (N_vis is small)
#ifndef XPR_IPT64
#define XPR_IPT64 8
#endif
constexpr int IPT64 = XPR_IPT64;            // supertile-word passes: 2048 words per tile
constexpr int PERSIST_CTAS = 148 * 4;       // upper bound of the persistent grids
constexpr int ST_SHIFT = 3, ST_EDGE = 1 << ST_SHIFT, ST_BINS = ST_EDGE * ST_EDGE;   // supertile: 8 x 8 tiles, 64 bins
constexpr int CHUNK = 256;                  // words of a supertile segment per final_kernel chunk (= its block size)
constexpr int CHUNK_WARPS = CHUNK / 32;

constexpr uint32_t FLAG_PARTIAL = 1u << 30, FLAG_INCLUSIVE = 2u << 30, FLAG_MASK = 3u << 30, VALUE_MASK = ~FLAG_MASK;
constexpr unsigned long long SFLAG_PARTIAL = 1ull << 62, SFLAG_INCLUSIVE = 2ull << 62, SFLAG_MASK = 3ull << 62;
constexpr unsigned long long FIELD_MAX = (1ull << 31) - 1;   // rank_scan packs two saturating 31-bit sums in one status word

// Header at the start of the workspace (zeroed every call).  The byte offsets of the first six fields are part
// of the asynchronous contract of xpr.h ([0,8) result, [8,16) pairs written) and of pipeline.py's diagnostics.
struct Header {
    unsigned long long total_pairs;          // I, or the capacity that suffices when pair_capacity does not
    unsigned long long pairs_out;            // pairs in the sorted output: I if everything fits, else 0
    unsigned long long l1_total;             // supertile words (Gaussian, supertile)
    unsigned long long rows_total;           // (Gaussian, tile row) rows of the visible Gaussians
    unsigned long long rows_eff;             // rows_total if the row table fits pair_capacity, else 0
    unsigned long long cand_total;           // candidate pairs: sum of tile_count
    unsigned long long l1_eff;               // l1_total if two word buffers fit pair_capacity and the rows fit, else 0
    uint32_t n_vis;                          // visible Gaussians
    uint32_t n_chunks;                       // chunks of final_kernel
    uint32_t compact_ticket, scan_ticket, final_ticket, pad0;
    uint32_t sort_ticket[DEPTH_PASSES + MAX_TILE_PASSES];
    uint32_t pad[4];
    uint32_t hist[(DEPTH_PASSES + MAX_TILE_PASSES) * RADIX];   // global digit histograms
};

struct Layout {
    size_t header, scan_status, status32, status64, final_status, tile_diff, seg_cnt, zero_end, seg_start, chunk_start, vkey0,
        vidx0, vkey1, vidx1, keys_tmp, total;
};

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

inline int digit_passes_for(int64_t n) {   // 8-bit digits needed for ids 0 .. n-1, at least one
    int bits = 0;
    while (bits < 31 && ((int64_t)1 << bits) < n) ++bits;
    const int p = (bits + RADIX_BITS - 1) / RADIX_BITS;
    return p < 1 ? 1 : p;
}

// Sizes depend on (N, capacity, number of tiles) only: the supertile count is bounded by the tile count.
inline Layout make_layout(int64_t N, int64_t cap, int32_t num_tiles) {
    Layout L;
    size_t off = 0;
    const size_t n = (size_t)N, c = (size_t)cap, T = (size_t)num_tiles;
    const size_t scan_blocks = (n + SCAN_ITEMS - 1) / SCAN_ITEMS;
    L.header = off; off = align_up(off + sizeof(Header), 256);
    L.scan_status = off; off = align_up(off + 8 * 2 * (scan_blocks + 1), 256);      // compact + rank-scan chains
    const size_t tiles32 = (n + SORT_THREADS * IPT32 - 1) / (SORT_THREADS * IPT32);
    L.status32 = off; off = align_up(off + 4 * (size_t)RADIX * tiles32 * DEPTH_PASSES, 256);
    const size_t tiles64 = (c / 2 + SORT_THREADS * IPT64 - 1) / (SORT_THREADS * IPT64) + 1;
    L.status64 = off; off = align_up(off + 4 * (size_t)RADIX * tiles64 * (size_t)digit_passes_for((int64_t)T), 256);
    const size_t chunks = c / 2 / CHUNK + T + 2;                                     // sum over segments of ceil(len / CHUNK)
    L.final_status = off; off = align_up(off + 4 * (size_t)ST_BINS * chunks, 256);
    L.tile_diff = off; off = align_up(off + 4 * (T + 2), 256);
    L.seg_cnt = off; off = align_up(off + 4 * (T + 2), 256);
    L.zero_end = off;   // everything up to here is zeroed with one memset
    L.seg_start = off; off = align_up(off + 4 * (T + 2), 256);
    L.chunk_start = off; off = align_up(off + 4 * (T + 2), 256);
    L.vkey0 = off; off = align_up(off + 4 * n, 256);
    L.vidx0 = off; off = align_up(off + 4 * n, 256);
    L.vkey1 = off; off = align_up(off + 4 * n, 256);
    L.vidx1 = off; off = align_up(off + 4 * n, 256);
    L.keys_tmp = off; off = align_up(off + 8 * c + 256, 256);   // row table (4 B x rows) | sorted supertile words (8 B x <= c/2)
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

// Chained scan across blocks (decoupled look-back), executed by warp 0 of a ticketed block: publishes
// the block's total and returns (to every lane of warp 0) the sum of the totals of all earlier blocks.
// `block` is a ticket, so every predecessor is running or done (forward progress).
// PAIR: the 62-bit value holds two 31-bit sums (rows | supertile words << 31) that saturate at FIELD_MAX
// (saturating addition of non-negative numbers is associative; a saturated sum exceeds any legal capacity).
template <bool PAIR>
__device__ __forceinline__ unsigned long long chain_add(unsigned long long a, unsigned long long b) {
    if (!PAIR) return a + b;
    const unsigned long long lo = min((a & FIELD_MAX) + (b & FIELD_MAX), FIELD_MAX);
    const unsigned long long hi = min(((a >> 31) & FIELD_MAX) + ((b >> 31) & FIELD_MAX), FIELD_MAX);
    return lo | (hi << 31);
}

template <bool PAIR>
__device__ __forceinline__ unsigned long long chain_lookback(uint32_t block, unsigned long long btotal,
                                                             unsigned long long* __restrict__ status, int lane) {
    unsigned long long excl = 0;
    if (block == 0) {
        if (lane == 0) st_relaxed64(&status[0], SFLAG_INCLUSIVE | btotal);
        return 0;
    }
    if (lane == 0) st_relaxed64(&status[block], SFLAG_PARTIAL | btotal);
    int64_t top = (int64_t)block - 1;          // lane l inspects predecessor top - l
    while (true) {
        const int64_t t = top - lane;
        unsigned long long sv = SFLAG_INCLUSIVE;   // virtual predecessors before block 0: inclusive 0
        if (t >= 0) { do { sv = ld_relaxed64(&status[t]); } while ((sv & SFLAG_MASK) == 0); }
        const uint32_t incl_mask = __ballot_sync(0xffffffffu, (sv & SFLAG_MASK) == SFLAG_INCLUSIVE);
        const int first = incl_mask ? (__ffs(incl_mask) - 1) : 32;     // nearest inclusive predecessor
        unsigned long long v = (lane <= first) ? (sv & ~SFLAG_MASK) : 0ull;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = chain_add<PAIR>(v, __shfl_xor_sync(0xffffffffu, v, o));
        excl = chain_add<PAIR>(excl, v);
        if (incl_mask) break;
        top -= 32;
    }
    if (lane == 0) st_relaxed64(&status[block], SFLAG_INCLUSIVE | chain_add<PAIR>(excl, btotal));
    return excl;
}

// ---------------------------------------------------------------------------------------------
// compact: visible Gaussians in index order -> (depth bits, index), + depth-digit histograms.
// A block owns SCAN_ITEMS consecutive Gaussians; warp w owns 256 of them and reads them in 8 coalesced
// rounds, so the in-warp prefix is just ballots and popcounts.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SCAN_THREADS)
compact_kernel(int64_t N, const float* __restrict__ depth, const uint32_t* __restrict__ tcount,
               Header* __restrict__ hdr, unsigned long long* __restrict__ status, uint32_t* __restrict__ vkey,
               uint32_t* __restrict__ vidx) {
    pdl_entry();
    __shared__ uint32_t s_warp[SCAN_WARPS];
    __shared__ uint32_t s_hist[DEPTH_PASSES * RADIX];
    __shared__ uint32_t s_block;
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_block = atomicAdd(&hdr->compact_ticket, 1u);
    for (int b = tid; b < DEPTH_PASSES * RADIX; b += SCAN_THREADS) s_hist[b] = 0u;
    __syncthreads();
    const uint32_t block = s_block;
    const int64_t i0 = (int64_t)block * SCAN_ITEMS + warp * (32 * SCAN_ROUNDS) + lane;
    uint32_t tc[SCAN_ROUNDS], db[SCAN_ROUNDS];
#pragma unroll
    for (int r = 0; r < SCAN_ROUNDS; ++r) {
        const int64_t i = i0 + r * 32;
        tc[r] = (i < N) ? __ldg(tcount + i) : 0u;
        db[r] = (i < N) ? __float_as_uint(__ldg(depth + i)) : 0u;   // never-written for a culled Gaussian; unused then
    }
    uint32_t pos[SCAN_ROUNDS], wtotal = 0;
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int r = 0; r < SCAN_ROUNDS; ++r) {
        const uint32_t m = __ballot_sync(0xffffffffu, tc[r] != 0u);
        pos[r] = wtotal + (uint32_t)__popc(m & lt);
        wtotal += (uint32_t)__popc(m);
    }
    if (lane == 0) s_warp[warp] = wtotal;
    __syncthreads();
    uint32_t wbase = 0, btotal = 0;
#pragma unroll
    for (int w = 0; w < SCAN_WARPS; ++w) {
        const uint32_t v = s_warp[w];
        if (w < warp) wbase += v;
        btotal += v;
    }
    if (warp == 0) {
        const unsigned long long e = chain_lookback<false>(block, (unsigned long long)btotal, status, lane);
        if (lane == 0) s_base = e;
    }
#pragma unroll
    for (int r = 0; r < SCAN_ROUNDS; ++r) {
        if (tc[r] != 0u) {
#pragma unroll
            for (int d = 0; d < DEPTH_PASSES; ++d) atomicAdd(&s_hist[d * RADIX + ((db[r] >> (8 * d)) & 255u)], 1u);
        }
    }
    __syncthreads();
    const unsigned long long base = s_base;
#pragma unroll
    for (int r = 0; r < SCAN_ROUNDS; ++r) {
        if (tc[r] != 0u) {
            const unsigned long long p = base + wbase + pos[r];
            vkey[p] = db[r];
            vidx[p] = (uint32_t)(i0 + r * 32);
        }
    }
    if (tid == 0 && (int64_t)(block + 1) * SCAN_ITEMS >= N) hdr->n_vis = (uint32_t)(base + btotal);
    for (int b = tid; b < DEPTH_PASSES * RADIX; b += SCAN_THREADS) {
        const uint32_t v = s_hist[b];
        if (v) atomicAdd(&hdr->hist[b], v);
    }
}

// ---------------------------------------------------------------------------------------------
// onesweep digit pass.  MODE 0: 32-bit keys + 32-bit values (the depth passes on the Gaussians);
// MODE 1: 64-bit words supertile << 32 | rank, no value (the supertile pass).
// ---------------------------------------------------------------------------------------------
template <class KeyT, int IPT, bool HAS_VAL>
struct SortSmem {
    KeyT keys[SORT_THREADS * IPT];
    uint32_t vals[HAS_VAL ? SORT_THREADS * IPT : 1];
    uint32_t warp_hist[SORT_WARPS][RADIX];
    uint32_t bitmap[SORT_WARPS][RADIX];   // BITMAP ranking: bit l of bitmap[w][d] = lane l of warp w holds digit d
    uint32_t cta_excl[RADIX];     // exclusive digit offsets inside the tile
    uint32_t gbase[RADIX];        // global position of digit d's first key of this tile, minus cta_excl[d]
    uint32_t scan_tmp[SORT_WARPS];
    uint32_t tile_id;
};

// BITMAP = true: the peer mask of a lane (lanes of its warp holding the same digit) is built in shared
// memory: every lane ORs its bit into bitmap[warp][digit] and reads the word back -- 3 shared-memory
// instructions instead of 8 ballots x 5 ALU instructions; conflict-free when the digits of a warp are
// distinct (mantissa bytes, consecutive tile ids), 32-way serialised when they are all equal.
// false: match.any (fast when a warp holds few distinct digits: the high tile digit).
#ifndef XPR_LB
#define XPR_LB 4
#endif
constexpr int LB = XPR_LB;   // look-back loads in flight per digit thread
#ifndef XPR_LB_EARLY
#define XPR_LB_EARLY 0
#endif
// Decoupled look-back over earlier tiles by the thread that owns one digit: sums the published counts
// of the predecessors down to the nearest one whose inclusive prefix is known, then publishes its own.
__device__ __forceinline__ uint32_t look_back(uint32_t* my, uint32_t tile, uint32_t real_count) {
    uint32_t excl_prev = 0;
    if (tile != 0) {
        const uint32_t* p = my - RADIX;
        uint32_t remaining = tile;
        bool found = false;
        while (!found) {   // LB predecessors in flight per round; before tile 0: virtual inclusive 0
            uint32_t sv[LB];
#pragma unroll
            for (int k = 0; k < LB; ++k)
                sv[k] = ((uint32_t)k < remaining) ? ld_relaxed(p - k * RADIX) : FLAG_INCLUSIVE;
#pragma unroll
            for (int k = 0; k < LB; ++k) {
                if (found) break;
                while ((sv[k] & FLAG_MASK) == 0u) sv[k] = ld_relaxed(p - k * RADIX);
                excl_prev += sv[k] & VALUE_MASK;
                found = (sv[k] & FLAG_MASK) == FLAG_INCLUSIVE;
            }
            p -= LB * RADIX;
            remaining = (remaining > (uint32_t)LB) ? remaining - (uint32_t)LB : 0u;
        }
        st_relaxed(my, FLAG_INCLUSIVE | (excl_prev + real_count));
    }
    return excl_prev;
}

template <class KeyT, int IPT, bool BITMAP, int MODE>
__global__ void __launch_bounds__(SORT_THREADS, 4)
onesweep_kernel(const uint32_t* __restrict__ n_dev32, const unsigned long long* __restrict__ n_dev64, int shift,
                int hist_row, int ticket_row, const KeyT* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                KeyT* __restrict__ keys_out, uint32_t* __restrict__ vals_out, Header* __restrict__ hdr,
                uint32_t* __restrict__ status /* [tiles][RADIX] of this pass */) {
    pdl_entry();
    constexpr int TILE_KEYS = SORT_THREADS * IPT;
    constexpr bool HAS_VAL = (MODE != 1);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem<KeyT, IPT, HAS_VAL>& S = *reinterpret_cast<SortSmem<KeyT, IPT, HAS_VAL>*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t n = n_dev32 ? *n_dev32 : (uint32_t)*n_dev64;

    if (BITMAP) {
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) S.bitmap[w][tid] = 0u;
    }
    // global position of digit tid's first key: exclusive scan of the global histogram (same for every tile)
    uint32_t bin_base;
    {
        const uint32_t gh = hdr->hist[hist_row * RADIX + tid];
        uint32_t inc = gh;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t a = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += a;
        }
        if (lane == 31) S.scan_tmp[warp] = inc;
        __syncthreads();
        uint32_t pre = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w)
            if (w < warp) pre += S.scan_tmp[w];
        bin_base = pre + inc - gh;
    }

    while (true) {
        __syncthreads();                                                  // previous tile done with shared memory
        if (tid == 0) S.tile_id = atomicAdd(&hdr->sort_ticket[ticket_row], 1u);
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) S.warp_hist[w][tid] = 0u;    // SORT_THREADS == RADIX
        __syncthreads();
        const uint32_t tile = S.tile_id;
        if ((uint64_t)tile * TILE_KEYS >= n) break;                       // tickets exhausted
        const uint32_t tile_base = tile * (uint32_t)TILE_KEYS;
        const uint32_t tile_n = min((uint32_t)TILE_KEYS, n - tile_base);

        // warp-striped load: item `it` of lane l of warp w sits at tile_base + w*32*IPT + it*32 + l
        KeyT key[IPT];
        const uint32_t wofs = (uint32_t)warp * 32u * IPT + (uint32_t)lane;
#pragma unroll
        for (int it = 0; it < IPT; ++it) {
            const uint32_t loc = wofs + (uint32_t)it * 32u;
            key[it] = (loc < tile_n) ? keys_in[tile_base + loc]
                                     : ~(KeyT)0;    // padding: highest digit, ranks after every real key of the tile
        }
        // stable in-warp ranking: rank = #earlier items of this warp with the same digit
        uint16_t rank[IPT];
        const uint32_t lt_mask = (1u << lane) - 1u;
#pragma unroll
        for (int it = 0; it < IPT; ++it) {
            const uint32_t d = (uint32_t)(key[it] >> shift) & (RADIX - 1);
            uint32_t peers;
            if (BITMAP) {
                atomicOr(&S.bitmap[warp][d], 1u << lane);
                __syncwarp();
                peers = S.bitmap[warp][d];
                __syncwarp();                                // everyone has read before the leader clears the word
            } else {
                peers = __match_any_sync(0xffffffffu, d);
            }
            const uint32_t lt = peers & lt_mask;
            uint32_t prev = 0;
            if (lt == 0u) {                                  // lowest lane of the peer group
                prev = S.warp_hist[warp][d];
                S.warp_hist[warp][d] = prev + (uint32_t)__popc(peers);
                if (BITMAP) S.bitmap[warp][d] = 0u;          // left zero for the next item / tile
            }
            __syncwarp();
            prev = __shfl_sync(0xffffffffu, prev, __ffs(peers) - 1);
            rank[it] = (uint16_t)(prev + (uint32_t)__popc(lt));
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
        // block exclusive scan over digits of `count` -> cta_excl
        uint32_t inc_c = count;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t a = __shfl_up_sync(0xffffffffu, inc_c, o);
            if (lane >= o) inc_c += a;
        }
        if (lane == 31) S.scan_tmp[warp] = inc_c;
        // publish this tile's digit counts at once
        uint32_t* my = status + (size_t)tile * RADIX + tid;
        st_relaxed(my, (tile == 0 ? FLAG_INCLUSIVE : FLAG_PARTIAL) | real_count);
        uint32_t excl_prev = 0;
        if (XPR_LB_EARLY) excl_prev = look_back(my, tile, real_count);
        __syncthreads();
        uint32_t pre_c = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w)
            if (w < warp) pre_c += S.scan_tmp[w];
        const uint32_t excl_c = pre_c + inc_c - count;        // position of digit tid inside the tile
        S.cta_excl[tid] = excl_c;
        __syncthreads();
        // scatter into shared memory in tile-sorted order (values are loaded only now: fewer live registers)
#pragma unroll
        for (int it = 0; it < IPT; ++it) {
            const uint32_t d = (uint32_t)(key[it] >> shift) & (RADIX - 1);
            const uint32_t pos = S.cta_excl[d] + S.warp_hist[warp][d] + rank[it];
            S.keys[pos] = key[it];
            if constexpr (HAS_VAL) {
                const uint32_t loc = wofs + (uint32_t)it * 32u;
                S.vals[pos] = (loc < tile_n) ? vals_in[tile_base + loc] : 0u;
            }
        }
        if (!XPR_LB_EARLY) excl_prev = look_back(my, tile, real_count);
        S.gbase[tid] = bin_base + excl_prev - excl_c;
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
                if constexpr (HAS_VAL) vals_out[dst] = S.vals[p];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// rank_scan: chained scans over the visible Gaussians in rank (= depth, index) order (PAPER L123
// "prefix-sum of tile counts", taken on the two coarser units of this design):
//   row_base[rank] = rows of the earlier Gaussians (a row = the tiles one Gaussian covers in one tile row),
//   l1_off[rank]   = supertile words of the earlier Gaussians (one word per 8 x 8 supertile its rectangle touches),
// and the totals, the candidate-pair total and the capacity verdict for the two tables.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t supertiles_of(const int4 q) {   // rectangle [x, z) x [y, w) in tiles, non-empty
    return (uint32_t)((((q.z - 1) >> ST_SHIFT) - (q.x >> ST_SHIFT) + 1) * (((q.w - 1) >> ST_SHIFT) - (q.y >> ST_SHIFT) + 1));
}

__global__ void __launch_bounds__(SCAN_THREADS)
rank_scan_kernel(const uint32_t* __restrict__ vidx, const int4* __restrict__ rect, const uint32_t* __restrict__ tcount,
                 Header* __restrict__ hdr, unsigned long long* __restrict__ status, uint32_t* __restrict__ row_base,
                 uint32_t* __restrict__ l1_off, unsigned long long pair_capacity) {
    pdl_entry();
    __shared__ uint32_t s_warp[2][SCAN_WARPS];
    __shared__ uint32_t s_block;
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t n = hdr->n_vis;
    for (;;) {       // persistent: blocks of SCAN_ITEMS Gaussians are drawn from a ticket counter (= look-back order)
        __syncthreads();
        if (tid == 0) s_block = atomicAdd(&hdr->scan_ticket, 1u);
        __syncthreads();
        const uint32_t block = s_block;
        if ((uint64_t)block * SCAN_ITEMS >= n && block != 0) return;   // beyond the list: nobody waits on us
        const uint32_t s0 = block * (uint32_t)SCAN_ITEMS + (uint32_t)warp * (32 * SCAN_ROUNDS) + (uint32_t)lane;
        uint32_t vh[SCAN_ROUNDS], vc[SCAN_ROUNDS];
        unsigned long long cand = 0;                       // candidate pairs of this thread's Gaussians
#pragma unroll
        for (int r = 0; r < SCAN_ROUNDS; ++r) {
            const uint32_t s = s0 + r * 32;
            vh[r] = vc[r] = 0u;
            if (s < n) {
                const uint32_t g = __ldg(vidx + s);
                const int4 q = __ldg(rect + g);
                vh[r] = (uint32_t)(q.w - q.y);
                vc[r] = supertiles_of(q);
                cand += __ldg(tcount + g);
            }
        }
        uint32_t eh[SCAN_ROUNDS], ec[SCAN_ROUNDS], th = 0, tc = 0;
#pragma unroll
        for (int r = 0; r < SCAN_ROUNDS; ++r) {
            uint32_t ih = vh[r], ic = vc[r];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t a = __shfl_up_sync(0xffffffffu, ih, o), b = __shfl_up_sync(0xffffffffu, ic, o);
                if (lane >= o) { ih += a; ic += b; }
            }
            eh[r] = th + ih - vh[r]; ec[r] = tc + ic - vc[r];
            th += __shfl_sync(0xffffffffu, ih, 31); tc += __shfl_sync(0xffffffffu, ic, 31);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) cand += __shfl_xor_sync(0xffffffffu, cand, o);
        if (lane == 0 && cand) atomicAdd(&hdr->cand_total, cand);
        if (lane == 0) { s_warp[0][warp] = th; s_warp[1][warp] = tc; }
        __syncthreads();
        uint32_t wbh = 0, wbc = 0, bth = 0, btc = 0;
#pragma unroll
        for (int w = 0; w < SCAN_WARPS; ++w) {
            const uint32_t a = s_warp[0][w], b = s_warp[1][w];
            if (w < warp) { wbh += a; wbc += b; }
            bth += a; btc += b;
        }
        if (warp == 0) {    // a block holds at most 2048 * 2^15 rows: no overflow inside the block
            const unsigned long long e = chain_lookback<true>(block, (unsigned long long)bth | ((unsigned long long)btc << 31),
                                                              status, lane);
            if (lane == 0) s_base = e;
        }
        __syncthreads();
        const unsigned long long base = s_base;
        const unsigned long long base_h = base & FIELD_MAX, base_c = (base >> 31) & FIELD_MAX;
        const bool last_block = (uint64_t)(block + 1) * SCAN_ITEMS >= n;
#pragma unroll
        for (int r = 0; r < SCAN_ROUNDS; ++r) {
            const uint32_t s = s0 + r * 32;
            if (s < n) {
                row_base[s] = (uint32_t)(base_h + wbh + eh[r]);
                l1_off[s] = (uint32_t)(base_c + wbc + ec[r]);
            }
        }
        if (tid == 0 && last_block) {
            const unsigned long long rows = min(base_h + bth, FIELD_MAX), l1 = min(base_c + btc, FIELD_MAX);
            hdr->rows_total = rows;
            hdr->l1_total = l1;
            // the row table holds 4 bytes per row in half of the second pair buffer; the sorted supertile words 8 bytes
            // each in the other half
            const bool rows_ok = rows < pair_capacity;
            hdr->rows_eff = rows_ok ? rows : 0ull;
            hdr->l1_eff = (rows_ok && 2ull * l1 <= pair_capacity) ? l1 : 0ull;
        }
        if (last_block) return;
    }
}

// ---------------------------------------------------------------------------------------------
// rows: one thread per (Gaussian, tile row) row of the visible Gaussians in rank order.  Without tile_cull a
// row is the whole width of the rectangle.  With tile_cull ("Cull") it is the interval of tiles
// that pass tile_keep: the set {x : min_{y in row} q <= lnv} is an interval (q is convex), so the kernel
// estimates its two ends analytically (the ellipse {q = lnv} cut by the strip of the row: its extreme x, or its
// intersection with the strip's edges) and then settles each end with the exact per-tile predicate tile_keep --
// the decision that defines the result (bit-identical to the oracle's) -- stepping while the predicate disagrees.
// ---------------------------------------------------------------------------------------------
// tile_cull of XPR-3DGS ("Cull", Listing 1, A.1.1 L435) for the tiles of ONE tile row: operator()(tx) is
// true when the pair (Gaussian, tile (tx, ty)) survives, i.e. unless min over the hull of the tile's pixel centres of
// 1/2 d^T K d exceeds lnv = ln(o / alpha_thresh) by more than the conservative margin.  Evaluation order and margin are
// reading C8 of DESIGN.md; every operation is individually rounded (explicit _rn intrinsics: this file is compiled with
// FMA contraction).  The terms that depend on the row only (the y edges, the facing y edge's minimiser -B dy / A and its
// c term) are formed once in init(): the same operations on the same operands as a per-tile evaluation, hoisted.
struct RowKeep {
    float mx, my, B, C, lnv, hA, hC, y_lo, y_hi, dyE, dxE, cE;
    bool in_y;
    __device__ __forceinline__ void init(float mx_, float my_, float A, float B_, float C_, float lnv_, uint32_t ty) {
        const float ts = (float)TILE;
        mx = mx_; my = my_; B = B_; C = C_; lnv = lnv_;
        hA = __fmul_rn(0.5f, A); hC = __fmul_rn(0.5f, C);
        const float y0 = __fadd_rn(__fmul_rn(ts, (float)ty), 0.5f), y1 = __fsub_rn(__fadd_rn(__fmul_rn(ts, (float)ty), ts), 0.5f);
        in_y = (my >= y0) && (my <= y1);
        y_lo = __fsub_rn(y0, my); y_hi = __fsub_rn(y1, my);
        dyE = __fsub_rn((my < y0) ? y0 : y1, my);               // the facing y edge (used when !in_y)
        dxE = __fdiv_rn(-__fmul_rn(B, dyE), A);
        cE = __fmul_rn(__fmul_rn(hC, dyE), dyE);
    }
    __device__ __forceinline__ bool drop(float a, float b, float c) const {
        const float margin = 1.0f / 262144.0f;   // 2^-18
        const float q = __fadd_rn(__fadd_rn(a, b), c);
        const float mag = __fadd_rn(__fadd_rn(__fadd_rn(fabsf(a), fabsf(b)), fabsf(c)), lnv);
        return q > __fadd_rn(lnv, __fmul_rn(mag, margin));
    }
    __device__ __forceinline__ bool operator()(uint32_t tx) const {
        const float ts = (float)TILE;
        const float x0 = __fadd_rn(__fmul_rn(ts, (float)tx), 0.5f), x1 = __fsub_rn(__fadd_rn(__fmul_rn(ts, (float)tx), ts), 0.5f);
        const bool in_x = (mx >= x0) && (mx <= x1);
        // both facing edges are evaluated unconditionally and selected afterwards (the same operations on the same operands
        // as the branching form; an edge that does not face the mean is ignored): the lanes of a warp stay together
        bool drop_x, drop_y;
        {
            const float dx = __fsub_rn((mx < x0) ? x0 : x1, mx);
            const float bx = __fmul_rn(B, dx);
            float dy = __fdiv_rn(-bx, C);
            dy = (dy < y_lo) ? y_lo : dy; dy = (y_hi < dy) ? y_hi : dy;
            drop_x = drop(__fmul_rn(__fmul_rn(hA, dx), dx), __fmul_rn(bx, dy), __fmul_rn(__fmul_rn(hC, dy), dy));
        }
        {
            const float lo = __fsub_rn(x0, mx), hi = __fsub_rn(x1, mx);
            float dx = dxE;
            dx = (dx < lo) ? lo : dx; dx = (hi < dx) ? hi : dx;
            drop_y = drop(__fmul_rn(__fmul_rn(hA, dx), dx), __fmul_rn(__fmul_rn(B, dx), dyE), cE);
        }
        // kept inside both ranges; else dropped iff dropped by every facing edge
        return (in_x && in_y) || !((in_x || drop_x) && (in_y || drop_y));
    }
};

__device__ __forceinline__ float approx_sqrt(float x) {   // the interval estimate needs no exact rounding
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

constexpr int ROW_SMEM = 2048;     // tile rows whose first-tile counter is kept in shared memory
// XPR-LinPrim's tile_cull (Eq. 2; reading L6): the bound on the chord over the tile,
//   dt_upper = max(0, min over the 16 ordered slab pairs of h_i + h_j + max over the 4 corners of (m_i - m_j)),
// keeps the pair iff sigma dt_upper >= -log(1 - alpha_thresh).  rec = lin_rec of the primitive (20 floats).  Every
// operation individually rounded, order as the oracle's.  m_i - m_j is affine in the tile position, so the kept tiles
// are the intersection of half-planes: convex, one interval per tile row.
__device__ __forceinline__ bool lin_tile_keep(const float* __restrict__ rec, int tx, int ty, float req) {
    const float ts = (float)TILE, mx = rec[0], my = rec[1];
    const float x0 = __fsub_rn(__fadd_rn(__fmul_rn(ts, (float)tx), 0.5f), mx), x1 = __fsub_rn(__fadd_rn(__fadd_rn(__fmul_rn(ts, (float)tx), ts), 0.5f), mx);
    const float y0 = __fsub_rn(__fadd_rn(__fmul_rn(ts, (float)ty), 0.5f), my), y1 = __fsub_rn(__fadd_rn(__fadd_rn(__fmul_rn(ts, (float)ty), ts), 0.5f), my);
    float mc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float kx = rec[4 + 3 * i], ky = rec[5 + 3 * i];
        mc[i][0] = -__fmaf_rn(kx, x0, __fmul_rn(ky, y0)); mc[i][1] = -__fmaf_rn(kx, x1, __fmul_rn(ky, y0));
        mc[i][2] = -__fmaf_rn(kx, x0, __fmul_rn(ky, y1)); mc[i][3] = -__fmaf_rn(kx, x1, __fmul_rn(ky, y1));
    }
    float best = INFINITY;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            float d = __fsub_rn(mc[i][0], mc[j][0]);
#pragma unroll
            for (int c = 1; c < 4; ++c) d = fmaxf(d, __fsub_rn(mc[i][c], mc[j][c]));
            best = fminf(best, __fadd_rn(__fadd_rn(d, rec[6 + 3 * i]), rec[6 + 3 * j]));
        }
    const float dt_upper = fmaxf(0.0f, best);
    return !(__fmul_rn(rec[2], dt_upper) < req);
}

template <int CULL>
__global__ void __launch_bounds__(128)
rows_kernel(int TW, int TH, int TH_view, const uint32_t* __restrict__ vidx, const uint32_t* __restrict__ row_base,
            const int4* __restrict__ rect, const float2* __restrict__ mean2d, const float4* __restrict__ conic_opac,
            const float* __restrict__ lnv, const float* __restrict__ lin_rec, float lin_req,
            const Header* __restrict__ hdr, uint32_t* __restrict__ row_tab, int* __restrict__ tile_diff) {
    pdl_entry();
    // one thread per row (grid-stride, a warp takes 32 consecutive rows).  The Gaussian of a row is the last one
    // whose first row is <= row: the warp finds it for its first row with a cooperative 32-ary search in the
    // strictly increasing row_base (4 dependent loads for 10^6 Gaussians instead of 20), loads the next 32 bases
    // with one coalesced read -- the 32 rows of the warp cannot span more Gaussians -- and every lane finishes
    // with a 5-step search over those through shuffles.
    // every row is COUNTED (the difference array gives I even when the row table does not fit: the capacity
    // report of xpr.h), and stored only if the table fits; a saturated total means more rows than any capacity
    const unsigned long long rows_total = hdr->rows_total;
    const uint32_t n_rows = (rows_total >= FIELD_MAX) ? 0u : (uint32_t)rows_total, n_vis = hdr->n_vis;
    const bool store = hdr->rows_eff != 0ull;
    __shared__ int s_rowstart[ROW_SMEM];
    for (int y = threadIdx.x; y <= TH && y < ROW_SMEM; y += 128) s_rowstart[y] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    for (uint32_t wrow = (blockIdx.x * 128u + threadIdx.x) & ~31u; wrow < n_rows; wrow += gridDim.x * 128u) {
        uint32_t lo = 0, hi = n_vis;                 // first index whose base is > wrow lies in [lo, hi]
        while (hi > lo) {
            const uint32_t len = hi - lo, stride = (len + 31u) / 32u;
            const uint32_t probe = min(lo + ((uint32_t)lane + 1u) * stride - 1u, hi - 1u);
            const uint32_t b = __ballot_sync(0xffffffffu, __ldg(row_base + probe) > wrow);
            if (b == 0u) { lo = hi; break; }
            const uint32_t f = (uint32_t)__ffs(b) - 1u;
            hi = min(lo + (f + 1u) * stride - 1u, hi - 1u);
            lo = lo + f * stride;
        }
        const uint32_t s0 = lo - 1u;                  // Gaussian of the warp's first row (row_base[0] == 0 <= wrow)
        const uint32_t rb = (s0 + (uint32_t)lane < n_vis) ? __ldg(row_base + s0 + lane) : 0xffffffffu;
        const uint32_t row = wrow + (uint32_t)lane;
        uint32_t k = 0;                               // last l in [0, 32) with row_base[s0 + l] <= row (l = 0 qualifies)
#pragma unroll
        for (int step = 16; step > 0; step >>= 1) {
            const uint32_t v = __shfl_sync(0xffffffffu, rb, (int)(k + step) & 31);
            if (k + step < 32u && v <= row) k += step;
        }
        if (row >= n_rows) continue;
        const uint32_t s = s0 + k;
        const uint32_t g = vidx[s];
        const int4 r = rect[g];
        const int ty = r.y + (int)(row - row_base[s]);
        float mx = 0.f, my = 0.f, A = 0.f, B = 0.f, C = 0.f, L = 0.f, ext = 0.f, det = 0.f;
        if (CULL == 1) {
            const float2 m = mean2d[g]; const float4 co = conic_opac[g];
            mx = m.x; my = m.y; A = co.x; B = co.y; C = co.z; L = lnv[g];
            det = A * C - B * B;
            ext = approx_sqrt(fmaxf(__fdividef(2.0f * L * C, det), 0.0f));   // half-width of the ellipse {q = L} in x
        }
        int xa = r.x, xb = r.z;                                 // kept tiles of this row: [xa, xb)
        if (CULL == 2) {
            // LinPrim: the kept tiles of the row are an interval (convexity above): its first and last tile by the exact predicate
            // (one interval [a, b) inside [xa, xb)).  The tile under the projected centre is kept whenever the row has a
            // kept tile near the centre column: from such a seed both ends are found by bisection (the predicate is
            // monotone on either side of a kept tile), O(log w) evaluations of the 64-term bound instead of one per
            // dropped tile; without a kept seed (rows far from the centre of a slanted primitive) the row is shrunk
            // from both ends tile by tile.  Either way the predicate alone decides: the result is the oracle's.
            const float* rec = lin_rec + 20 * (size_t)g;
            const int seed = min(max((int)floorf(rec[0] * (1.0f / (float)TILE)), xa), xb - 1);
            if (lin_tile_keep(rec, seed, ty, lin_req)) {
                int lo = xa, hi = seed;                    // first kept tile in [xa, seed]: keep(hi) holds
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (lin_tile_keep(rec, mid, ty, lin_req)) hi = mid; else lo = mid + 1;
                }
                xa = hi;
                lo = seed; hi = xb - 1;                    // last kept tile in [seed, xb - 1]: keep(lo) holds
                while (lo < hi) {
                    const int mid = (lo + hi + 1) >> 1;
                    if (lin_tile_keep(rec, mid, ty, lin_req)) lo = mid; else hi = mid - 1;
                }
                xb = lo + 1;
            } else {
                while (xa < xb && !lin_tile_keep(rec, xa, ty, lin_req)) ++xa;
                while (xb > xa && !lin_tile_keep(rec, xb - 1, ty, lin_req)) --xb;
            }
        }
        if (CULL == 1) {
            const int tyv = ty % TH_view;              // batch of views: the tile rows of view v are offset by v * TH_view
            RowKeep keep;
            keep.init(mx, my, A, B, C, L, (uint32_t)tyv);
            // estimate: x extent of {q <= L} over dy in [lo, hi] (pixel-centre hull of the row)
            const float lo = (float)(TILE * tyv) + 0.5f - my, hi = (float)(TILE * tyv + TILE) - 0.5f - my;
            float left = 1e30f, right = -1e30f;
            const float rA = __fdividef(1.0f, A);
            const float dy_ext = __fdividef(B * ext, C);        // dy at the ellipse's extreme x: -B dx / C, dx = -+ext
            if (dy_ext >= lo && dy_ext <= hi) left = -ext;
            if (-dy_ext >= lo && -dy_ext <= hi) right = ext;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const float c = e ? hi : lo;
                const float disc = 2.0f * A * L - det * c * c;  // roots of q(dx, c) = L
                if (disc >= 0.0f) {
                    const float sq = approx_sqrt(disc), mid = -B * c;
                    left = fminf(left, (mid - sq) * rA); right = fmaxf(right, (mid + sq) * rA);
                }
            }
            if (lo <= 0.0f && hi >= 0.0f) { left = fminf(left, 0.0f); right = fmaxf(right, 0.0f); }   // the mean's row
            // q_min over the row's tiles is convex in x, so if any tile is kept the one nearest the row's minimiser x* is:
            // x* = mx when the mean lies in the row's strip, else mx - B c / A with c the strip edge nearest the mean
            const float cm = (lo <= 0.0f && hi >= 0.0f) ? 0.0f : ((lo > 0.0f) ? lo : hi);
            const int tc = max(r.x, min(r.z - 1, (int)floorf((mx - B * cm * rA) * (1.0f / (float)TILE))));
            // The two ends are settled with the exact predicate by ONE loop around ONE evaluation: every lane carries a
            // small state (which end, which direction, the candidate tile), so that the lanes of a warp evaluate their
            // candidates together whatever paths their rows take (separate loops per case serialise the warp and repeat
            // the predicate's code a dozen times).  Typical row: 4 evaluations (keep(a), !keep(a - 1), keep(b - 1), !keep(b)).
            //   L0 first probe of the left end · LOUT stepping outwards while kept · LIN stepping inwards until kept
            //   R0 / ROUT / RIN the same for the right end · C0 C1 C2 the estimate saw nothing: probe the tile nearest x*
            //   and its two neighbours (rounding of x*), then grow from there
            enum { L0, LOUT, LIN, R0, ROUT, RIN, C0, C1, C2, DONE };
            int st, cand, a = r.x, b = r.x, xe = r.z;
            if (left <= right) {
                const int a0 = max(r.x, min(r.z - 1, (int)floorf((mx + left - ((float)TILE - 0.5f)) * (1.0f / (float)TILE)) + 1));
                xe = max(a0, min(r.z - 1, (int)floorf((mx + right - 0.5f) * (1.0f / (float)TILE)))) + 1;   // exclusive
                st = L0; cand = a0;
            } else { st = C0; cand = tc; }
            while (st != DONE) {
                const bool k = keep((uint32_t)cand);
                const bool was_centre = st >= C0;
                bool to_right = false, to_centre = false, empty = false;
                if (st == L0 || st == LOUT || was_centre) {
                    if (k) {
                        a = cand;
                        if (was_centre) xe = cand + 1;
                        if (cand > r.x) { st = LOUT; cand = cand - 1; } else to_right = true;
                    } else if (st == LOUT) to_right = true;
                    else if (st == L0) { if (cand + 1 < xe) { st = LIN; cand = cand + 1; } else to_centre = true; }
                    else if (st == C0 && tc > r.x) { st = C1; cand = tc - 1; }
                    else if (st != C2 && tc + 1 < r.z) { st = C2; cand = tc + 1; }
                    else empty = true;
                } else if (st == LIN) {
                    if (k) { a = cand; to_right = true; }
                    else if (cand + 1 < xe) cand = cand + 1;
                    else to_centre = true;
                } else if (st == R0 || st == ROUT) {
                    if (k) { b = cand + 1; if (b < r.z) { st = ROUT; cand = b; } else st = DONE; }
                    else if (st == ROUT) st = DONE;
                    else if (cand - 1 > a) { st = RIN; cand = cand - 1; }
                    else { b = a + 1; st = DONE; }
                } else {   // RIN
                    if (k) { b = cand + 1; st = DONE; }
                    else if (cand - 1 > a) cand = cand - 1;
                    else { b = a + 1; st = DONE; }
                }
                if (to_right) { st = R0; cand = max(xe - 1, a); }
                if (to_centre) { st = C0; cand = tc; }
                if (empty) { a = b = r.x; st = DONE; }
            }
            xa = a; xb = b;
        }
        // the row as (first column, length); its tiles ty TW + xa ... are consecutive ids: +1 where the run starts,
        // -1 behind its end -- the running sum of the array is the number of pairs of every tile
        if (store) row_tab[row] = (uint32_t)xa | ((uint32_t)(xb - xa) << 16);
        if (xb > xa) {
            // the first tile of a tile row is the hot address (every Gaussian clipped by the left image edge starts
            // there, every one clipped by the right edge ends at the next row's first tile): those go to shared memory
            const int t0 = ty * TW;
            if (xa == 0 && ty < ROW_SMEM) atomicAdd(&s_rowstart[ty], 1); else atomicAdd(tile_diff + t0 + xa, 1);
            if (xb == TW && ty + 1 < ROW_SMEM) atomicAdd(&s_rowstart[ty + 1], -1); else atomicAdd(tile_diff + t0 + xb, -1);
        }
    }
    __syncthreads();
    for (int y = threadIdx.x; y <= TH && y < ROW_SMEM; y += 128) {
        const int v = s_rowstart[y];
        if (v) atomicAdd(tile_diff + y * TW, v);
    }
}

// ---------------------------------------------------------------------------------------------
// l1_emit: one thread per visible Gaussian (rank order): one word supertile << 32 | rank per supertile its
// rectangle touches, row-major inside the rectangle, at l1_off[rank] -- emission in rank order, so the stable
// sort by supertile leaves every segment in rank order.  Also the digit histograms of the supertile ids (for
// the onesweep passes) and the number of words of every supertile (the segments).
// ---------------------------------------------------------------------------------------------
constexpr int SEG_SMEM = 4096;              // supertile counters kept in shared memory (larger images: global atomics)
template <int PASSES>
__global__ void __launch_bounds__(256)
l1_emit_kernel(int STW, uint32_t ST, const uint32_t* __restrict__ vidx, const int4* __restrict__ rect,
               const uint32_t* __restrict__ l1_off, Header* __restrict__ hdr, uint64_t* __restrict__ words,
               uint32_t* __restrict__ seg_cnt) {
    pdl_entry();
    __shared__ uint32_t s_hist[PASSES * RADIX];
    __shared__ uint32_t s_seg[SEG_SMEM];
    if (hdr->l1_eff == 0ull) return;                    // nothing visible, or the tables do not fit
    const uint32_t n_vis = hdr->n_vis;
    const bool seg_shared = ST <= (uint32_t)SEG_SMEM;   // a few hundred addresses: global atomics would serialise on them
    for (int b = threadIdx.x; b < PASSES * RADIX; b += 256) s_hist[b] = 0u;
    if (seg_shared) for (uint32_t b = threadIdx.x; b < ST; b += 256) s_seg[b] = 0u;
    __syncthreads();
    for (uint32_t r = blockIdx.x * 256u + threadIdx.x; r < n_vis; r += gridDim.x * 256u) {
        const int4 q = __ldg(rect + __ldg(vidx + r));
        const int sx0 = q.x >> ST_SHIFT, sx1 = ((q.z - 1) >> ST_SHIFT) + 1;
        const int sy0 = q.y >> ST_SHIFT, sy1 = ((q.w - 1) >> ST_SHIFT) + 1;
        uint32_t off = __ldg(l1_off + r);
        for (int sy = sy0; sy < sy1; ++sy)
            for (int sx = sx0; sx < sx1; ++sx) {
                const uint32_t sid = (uint32_t)(sy * STW + sx);
                words[off++] = ((uint64_t)sid << 32) | (uint64_t)r;
                if (seg_shared) atomicAdd(&s_seg[sid], 1u); else atomicAdd(seg_cnt + sid, 1u);
#pragma unroll
                for (int d = 0; d < PASSES; ++d) atomicAdd(&s_hist[d * RADIX + ((sid >> (8 * d)) & 255u)], 1u);
            }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < PASSES * RADIX; b += 256) {
        const uint32_t v = s_hist[b];
        if (v) atomicAdd(&hdr->hist[DEPTH_PASSES * RADIX + b], v);
    }
    if (seg_shared)
        for (uint32_t b = threadIdx.x; b < ST; b += 256) {
            const uint32_t v = s_seg[b];
            if (v) atomicAdd(seg_cnt + b, v);
        }
}

// ---------------------------------------------------------------------------------------------
// tile_scan (one CTA): "identify bounds" without the pairs.  The running sum of the rows'
// difference array is the number of pairs of every tile, its exclusive prefix the tile's first position:
// tile_ranges[t] = (start, end), (0, 0) for an empty tile; I = the grand total.  Then the capacity verdict
// (xpr.h): the call needs pair_capacity >= max(I, rows + 1, 2 x supertile words).  If it fits, the supertile
// segments (exclusive prefix of the per-supertile word counts) and the chunk table of final_kernel.
// ---------------------------------------------------------------------------------------------
constexpr int TS_THREADS = 1024;

__device__ __forceinline__ uint32_t block_scan_incl(uint32_t v, uint32_t* s_warp, uint32_t& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t a = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += a;
    }
    __syncthreads();                       // s_warp free (previous use)
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint32_t pre = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < TS_THREADS / 32; ++w) {
        const uint32_t a = s_warp[w];
        if (w < warp) pre += a;
        tot += a;
    }
    total = tot;
    return pre + incl;
}

__global__ void __launch_bounds__(TS_THREADS)
tile_scan_kernel(uint32_t T, uint32_t ST, unsigned long long pair_capacity, const int* __restrict__ tile_diff,
                 const uint32_t* __restrict__ seg_cnt, uint2* __restrict__ ranges, uint32_t* __restrict__ seg_start,
                 uint32_t* __restrict__ chunk_start, Header* __restrict__ hdr) {
    pdl_entry();
    __shared__ uint32_t s_warp[TS_THREADS / 32];
    const uint32_t tid = threadIdx.x;
    // per-tile counts (running sum of the differences) and bases (exclusive prefix of the counts): a thread owns
    // `per` consecutive tiles, so each of the two prefix sums is a local loop, one block scan and a local loop
    __shared__ unsigned long long s_wtot[TS_THREADS / 32];
    __shared__ unsigned long long s_total;
    const int lane = tid & 31, warp = tid >> 5;
    const uint32_t per = (T + TS_THREADS - 1) / TS_THREADS;
    const uint32_t t_lo = min(tid * per, T), t_hi = min(t_lo + per, T);
    uint32_t dsum = 0;
    for (uint32_t t = t_lo; t < t_hi; ++t) dsum += (uint32_t)tile_diff[t];          // two's complement: exact mod 2^32
    uint32_t tot_d;
    const uint32_t cnt0 = block_scan_incl(dsum, s_warp, tot_d) - dsum;             // running sum before my first tile
    uint32_t cnt = cnt0;
    unsigned long long csum = 0;                                                    // pairs of my tiles
    for (uint32_t t = t_lo; t < t_hi; ++t) { cnt += (uint32_t)tile_diff[t]; csum += cnt; }
    unsigned long long base;                                                        // pairs of all earlier tiles (64-bit scan)
    {
        unsigned long long incl = csum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long a = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += a;
        }
        if (lane == 31) s_wtot[warp] = incl;
        __syncthreads();
        unsigned long long pre = 0, tot = 0;
#pragma unroll
        for (int w = 0; w < TS_THREADS / 32; ++w) {
            const unsigned long long a = s_wtot[w];
            if (w < warp) pre += a;
            tot += a;
        }
        base = pre + incl - csum;
        if (tid == 0) s_total = tot;
        __syncthreads();
    }
    const unsigned long long carry_base = s_total;
    cnt = cnt0;
    for (uint32_t t = t_lo; t < t_hi; ++t) {
        cnt += (uint32_t)tile_diff[t];
        // positions beyond 2^32 cannot occur for a count that fits the capacity; the ranges are zeroed below otherwise
        ranges[t] = cnt ? make_uint2((uint32_t)base, (uint32_t)(base + cnt)) : make_uint2(0u, 0u);
        base += cnt;
    }
    const unsigned long long I = carry_base;
    const unsigned long long rows = hdr->rows_total, l1 = hdr->l1_total;
    const bool ok = I <= pair_capacity && (rows == 0ull || hdr->rows_eff != 0ull) && (l1 == 0ull || hdr->l1_eff != 0ull);
    if (!ok) {
        for (uint32_t t = tid; t < T; t += TS_THREADS) ranges[t] = make_uint2(0u, 0u);
        if (tid == 0) {
            unsigned long long need = I;
            if (rows + 1 > need) need = rows + 1;
            if (2 * l1 > need) need = 2 * l1;
            hdr->total_pairs = need;
            hdr->pairs_out = 0ull;
            hdr->n_chunks = 0u;
        }
        return;
    }
    // supertile segments and chunks
    uint32_t carry_s = 0, carry_c = 0;
    for (uint32_t s0 = 0; s0 < ST; s0 += TS_THREADS) {
        const uint32_t s = s0 + tid;
        const uint32_t n = (s < ST) ? seg_cnt[s] : 0u;
        const uint32_t ch = (n + CHUNK - 1) / CHUNK;
        uint32_t tot_n, tot_ch;
        const uint32_t in = block_scan_incl(n, s_warp, tot_n);
        const uint32_t ic = block_scan_incl(ch, s_warp, tot_ch);
        if (s < ST) { seg_start[s] = carry_s + in - n; chunk_start[s] = carry_c + ic - ch; }
        carry_s += tot_n;
        carry_c += tot_ch;
    }
    if (tid == 0) {
        seg_start[ST] = carry_s;
        chunk_start[ST] = carry_c;
        hdr->total_pairs = I;
        hdr->pairs_out = I;
        hdr->n_chunks = carry_c;
    }
}

// ---------------------------------------------------------------------------------------------
// final: replicate + assign tile id + (the tile digits of the) sort in one pass.  A chunk is up to
// CHUNK consecutive words of ONE supertile's segment (words in rank order); thread i first owns word i:
//   1. its Gaussian's rows inside the supertile (row table) -> 64-bit mask of the tiles it covers there;
//   2. per warp and per tile bit present in the warp: ballot -> the column of the bit (which lanes cover the
//      tile) and its population count;
//   3. per (chunk, bit): exclusive prefix over the warps, total published, decoupled look-back over the earlier
//      chunks of the segment (the chunk index is a ticket: every predecessor is running or done);
//   4. the warp walks the bits present in it once more: for a fixed bit the covering lanes write consecutive
//      positions, tile start + pairs of earlier chunks + pairs of earlier warps + covering lanes before me (popcount
//      of the saved column below the lane): key = tile << 32 | depth bits, value = Gaussian index.
//      (Measured alternatives, config 5 / config 3, this variant 380 / 48 us: every lane walking its own bits, fewest
//      instructions but scattered stores, 627 / 50 us; one pair per thread in output order, fully coalesced, with a
//      select of the k-th set bit per pair 410 / 43 us, with a byte table of word numbers in shared memory 464 / 56 us;
//      staging key and value of the pairs in shared memory in rounds 655 / 74 us.)
// Within a tile the pairs are in rank = (depth, index) order: the stable sort by (tile, depth).
// ---------------------------------------------------------------------------------------------
#ifndef XPR_FINAL_LB
#define XPR_FINAL_LB 4
#endif
// Transpose of a 32 x 32 bit matrix held one row per lane: on return lane j holds column j (bit i = row i's bit j).
// Five exchange steps; in step s the lanes without bit s keep their columns without bit s and take those of their partner
// into the upper positions, the lanes with bit s do the opposite.
__device__ __forceinline__ uint32_t warp_transpose32(uint32_t x, int lane) {
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        const uint32_t m = (s == 16) ? 0x0000ffffu : (s == 8) ? 0x00ff00ffu : (s == 4) ? 0x0f0f0f0fu : (s == 2) ? 0x33333333u : 0x55555555u;
        const uint32_t t = __shfl_xor_sync(0xffffffffu, x, s);
        x = (lane & s) ? ((x & ~m) | ((t & ~m) >> s)) : ((x & m) | ((t & m) << s));
    }
    return x;
}

__global__ void __launch_bounds__(CHUNK)
final_kernel(int TW, int TH, int STW, uint32_t ST, const uint64_t* __restrict__ words,
             const uint32_t* __restrict__ seg_start, const uint32_t* __restrict__ chunk_start,
             const uint32_t* __restrict__ vkey, const uint32_t* __restrict__ vidx, const int4* __restrict__ rect,
             const uint32_t* __restrict__ row_base, const uint32_t* __restrict__ row_tab,
             const uint2* __restrict__ ranges, Header* __restrict__ hdr, uint32_t* __restrict__ status,
             uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out) {
    pdl_entry();
    __shared__ uint32_t s_cnt[CHUNK_WARPS][ST_BINS];    // per warp: covering lanes, then exclusive prefix over warps
    __shared__ uint32_t s_base[ST_BINS];                // global position of the chunk's first pair of every bit
    __shared__ uint32_t s_chunk, s_seg, s_seg_c0;       // ticket; supertile of the chunk; first chunk of that supertile
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t n_chunks = hdr->n_chunks;
    uint32_t seg = 0;                                   // tickets grow: the search resumes where the last one ended
    while (true) {
        __syncthreads();                                // previous chunk done with the shared arrays
        if (tid == 0) s_chunk = atomicAdd(&hdr->final_ticket, 1u);
        __syncthreads();
        const uint32_t chunk = s_chunk;
        if (chunk >= n_chunks) break;
        if (warp == 0) {
            // supertile of the chunk: last s with chunk_start[s] <= chunk.  Galloping 32-ary search from the
            // previous answer (chunks of one CTA are increasing and mostly in the same or a near supertile)
            uint32_t lo = seg;                          // chunk_start[lo] <= chunk
            while (true) {
                const uint32_t probe = min(lo + 1u + (uint32_t)lane, ST);
                const uint32_t v = __ldg(chunk_start + probe);
                const uint32_t b = __ballot_sync(0xffffffffu, v > chunk);     // chunk_start[ST] = n_chunks > chunk
                if (b) { lo = lo + (uint32_t)__ffs(b) - 1u; break; }
                lo += 32u;
            }
            if (lane == 0) { s_seg = lo; s_seg_c0 = __ldg(chunk_start + lo); }
        }
        __syncthreads();
        seg = s_seg;
        const uint32_t c0 = s_seg_c0;
        const uint32_t w0 = __ldg(seg_start + seg) + (chunk - c0) * (uint32_t)CHUNK, w1 = __ldg(seg_start + seg + 1);
        const uint32_t n = min((uint32_t)CHUNK, w1 - w0);
        const int sx = (int)(seg % (uint32_t)STW), sy = (int)(seg / (uint32_t)STW);
        const int tx0 = sx << ST_SHIFT, ty0 = sy << ST_SHIFT;
        // 1. mask of my Gaussian's tiles inside the supertile
        uint32_t m_lo = 0, m_hi = 0, g = 0, dbits = 0;
        if ((uint32_t)tid < n) {
            const uint32_t r = (uint32_t)words[w0 + tid];
            g = __ldg(vidx + r);
            dbits = __ldg(vkey + r);
            const int4 q = __ldg(rect + g);
            const uint32_t rb = __ldg(row_base + r);
            const int ya = max(q.y, ty0), yb = min(q.w, ty0 + ST_EDGE);
            uint32_t e[ST_EDGE];
#pragma unroll
            for (int k = 0; k < ST_EDGE; ++k) {
                const int ty = ty0 + k;
                e[k] = (ty >= ya && ty < yb) ? __ldg(row_tab + rb + (uint32_t)(ty - q.y)) : 0u;
            }
#pragma unroll
            for (int k = 0; k < ST_EDGE; ++k) {
                const int xa = (int)(e[k] & 0xffffu), xb = xa + (int)(e[k] >> 16);
                const int a = max(xa, tx0) - tx0, b = min(xb, tx0 + ST_EDGE) - tx0;
                const uint32_t bits = (b > a) ? ((0xffu >> (ST_EDGE - b)) & (0xffu << a)) & 0xffu : 0u;
                if (k < 4) m_lo |= bits << (8 * k); else m_hi |= bits << (8 * (k - 4));
            }
        }
        // 2. per warp: the column (which lanes cover the bit's tile) and the count of every bit.  The 32 masks of a warp are
        //    a 32 x 64 bit matrix; its transpose -- lane b ends with columns b and 32 + b -- takes 5 exchange steps per
        //    32 x 32 half (a ballot per bit present was 64 iterations of ~8 instructions)
        const uint32_t u_lo = __reduce_or_sync(0xffffffffu, m_lo), u_hi = __reduce_or_sync(0xffffffffu, m_hi);
        const uint32_t c_lo = warp_transpose32(m_lo, lane), c_hi = warp_transpose32(m_hi, lane);
        s_cnt[warp][lane] = (uint32_t)__popc(c_lo);
        s_cnt[warp][32 + lane] = (uint32_t)__popc(c_hi);
        __syncthreads();
        // 3. per bit: prefix over the warps, look-back over the earlier chunks of this segment
        if (tid < ST_BINS) {
            uint32_t count = 0;
#pragma unroll
            for (int w = 0; w < CHUNK_WARPS; ++w) {
                const uint32_t v = s_cnt[w][tid];
                s_cnt[w][tid] = count;
                count += v;
            }
            uint32_t* my = status + (size_t)chunk * ST_BINS + tid;
            const bool first = chunk == c0;
            st_relaxed(my, (first ? FLAG_INCLUSIVE : FLAG_PARTIAL) | count);
            uint32_t excl_prev = 0;
            if (!first) {
                const uint32_t* p = my - ST_BINS;
                uint32_t remaining = chunk - c0;
                bool found = false;
                while (!found) {
                    uint32_t sv[XPR_FINAL_LB];
#pragma unroll
                    for (int k = 0; k < XPR_FINAL_LB; ++k)
                        sv[k] = ((uint32_t)k < remaining) ? ld_relaxed(p - k * ST_BINS) : FLAG_INCLUSIVE;
#pragma unroll
                    for (int k = 0; k < XPR_FINAL_LB; ++k) {
                        if (found) break;
                        while ((sv[k] & FLAG_MASK) == 0u) sv[k] = ld_relaxed(p - k * ST_BINS);
                        excl_prev += sv[k] & VALUE_MASK;
                        found = (sv[k] & FLAG_MASK) == FLAG_INCLUSIVE;
                    }
                    p -= XPR_FINAL_LB * ST_BINS;
                    remaining = (remaining > (uint32_t)XPR_FINAL_LB) ? remaining - (uint32_t)XPR_FINAL_LB : 0u;
                }
                st_relaxed(my, FLAG_INCLUSIVE | (excl_prev + count));
            }
            const int tx = tx0 + (tid & (ST_EDGE - 1)), ty = ty0 + (tid >> ST_SHIFT);
            const bool inside = tx < TW && ty < TH;
            s_base[tid] = (inside ? ranges[ty * TW + tx].x : 0u) + excl_prev;
        }
        __syncthreads();
        // 4. scatter: the warp walks the 64 bits once more (unrolled; a bit absent from the whole warp is skipped); for a
        //    fixed bit the covering lanes (the column of step 2, still in lane b's register) write consecutive positions:
        //    tile start + pairs of earlier chunks + pairs of earlier warps + covering lanes before me.  Column, first
        //    position and tile id of bit b are broadcast from lane b by shuffles (the loop over __ffs with three
        //    shared-memory reads per bit took 30 instructions per bit: 76 % of the kernel's instructions)
        {
            const uint32_t p_lo = s_cnt[warp][lane] + s_base[lane], p_hi = s_cnt[warp][lane + 32] + s_base[lane + 32];
            const uint32_t t_lo = (uint32_t)((ty0 + (lane >> ST_SHIFT)) * TW + tx0 + (lane & (ST_EDGE - 1)));
            const uint32_t t_hi = t_lo + (uint32_t)(4 * TW);
            const uint32_t lt = (1u << lane) - 1u;
            const uint64_t dkey = (uint64_t)dbits;
#pragma unroll
            for (int b = 0; b < 32; ++b) {
                if (!((u_lo >> b) & 1u)) continue;                       // warp-uniform
                const uint32_t col = __shfl_sync(0xffffffffu, c_lo, b), p0 = __shfl_sync(0xffffffffu, p_lo, b);
                const uint32_t tl = __shfl_sync(0xffffffffu, t_lo, b);
                if ((m_lo >> b) & 1u) {
                    const uint32_t pos = p0 + (uint32_t)__popc(col & lt);
                    keys_out[pos] = ((uint64_t)tl << 32) | dkey;
                    vals_out[pos] = g;
                }
            }
#pragma unroll
            for (int b = 0; b < 32; ++b) {
                if (!((u_hi >> b) & 1u)) continue;
                const uint32_t col = __shfl_sync(0xffffffffu, c_hi, b), p0 = __shfl_sync(0xffffffffu, p_hi, b);
                const uint32_t tl = __shfl_sync(0xffffffffu, t_hi, b);
                if ((m_hi >> b) & 1u) {
                    const uint32_t pos = p0 + (uint32_t)__popc(col & lt);
                    keys_out[pos] = ((uint64_t)tl << 32) | dkey;
                    vals_out[pos] = g;
                }
            }
        }
    }
}

// Scheduling aid for the compositing kernels (xpr_config.tile_order): the tile indices by decreasing list length,
// in 1024 length classes (counting sort, one CTA: T is a few thousand).  Heaviest tiles first means the last wave
// of a compositing launch is made of short tiles.
__global__ void __launch_bounds__(1024)
tile_order_kernel(const uint32_t* __restrict__ ranges, uint32_t T, uint32_t* __restrict__ order) {
    pdl_entry();
    __shared__ uint32_t s_cnt[1024];
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_shift;
    const uint32_t tid = threadIdx.x;
    uint32_t mx = 0;
    for (uint32_t t = tid; t < T; t += 1024) mx = max(mx, ranges[2 * t + 1] - ranges[2 * t]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((tid & 31) == 0) s_warp[tid >> 5] = mx;
    s_cnt[tid] = 0;
    __syncthreads();
    if (tid == 0) {
        uint32_t m = 0;
        for (int w = 0; w < 32; ++w) m = max(m, s_warp[w]);
        const int bits = 32 - __clz(m | 1u);
        s_shift = (uint32_t)max(0, bits - 10);
    }
    __syncthreads();
    const uint32_t shift = s_shift;
    for (uint32_t t = tid; t < T; t += 1024)      // class 0 = longest
        atomicAdd(&s_cnt[1023u - min(1023u, (ranges[2 * t + 1] - ranges[2 * t]) >> shift)], 1u);
    __syncthreads();
    // exclusive scan of the 1024 class counts
    const uint32_t c = s_cnt[tid];
    uint32_t incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if ((tid & 31) >= (uint32_t)o) incl += v;
    }
    if ((tid & 31) == 31) s_warp[tid >> 5] = incl;
    __syncthreads();
    if (tid < 32) {
        uint32_t w = s_warp[tid], wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, wi, o);
            if (tid >= (uint32_t)o) wi += v;
        }
        s_warp[tid] = wi - w;
    }
    __syncthreads();
    s_cnt[tid] = s_warp[tid >> 5] + incl - c;
    __syncthreads();
    for (uint32_t t = tid; t < T; t += 1024) {
        const uint32_t cls = 1023u - min(1023u, (ranges[2 * t + 1] - ranges[2 * t]) >> shift);
        order[atomicAdd(&s_cnt[cls], 1u)] = t;
    }
}

}  // namespace
}  // namespace xpr

using namespace xpr;

extern "C" int32_t xpr_bin_sort_workspace(int64_t N, int64_t pair_capacity, int32_t num_tiles, size_t* bytes) {
    if (!bytes || N < 0 || pair_capacity < 0 || pair_capacity >= (1LL << 30) || num_tiles <= 0)
        return XPR_ERR_INVALID_ARG;
    if (N >= (1LL << 30)) return XPR_ERR_UNSUPPORTED;      // the look-back status words carry 30-bit counts
    if (num_tiles > (1 << 24)) return XPR_ERR_UNSUPPORTED;
    *bytes = make_layout(N, pair_capacity, num_tiles).total;
    return XPR_OK;
}

template <class KeyT, int IPT, bool BITMAP, int MODE>
static cudaError_t launch_pass(unsigned tiles, cudaStream_t st, const uint32_t* n32, const unsigned long long* n64,
                               int shift, int row, const KeyT* kin, const uint32_t* vin, KeyT* kout, uint32_t* vout,
                               Header* hdr, uint32_t* status) {
    const size_t smem = sizeof(SortSmem<KeyT, IPT, MODE != 1>);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(onesweep_kernel<KeyT, IPT, BITMAP, MODE>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const unsigned grid = tiles < (unsigned)PERSIST_CTAS ? tiles : (unsigned)PERSIST_CTAS;
    return launch_k(true, onesweep_kernel<KeyT, IPT, BITMAP, MODE>, dim3(grid), dim3(SORT_THREADS), smem, st, n32, n64, shift,
                    row, row, kin, vin, kout, vout, hdr, status);
}

// Common body of xpr_bin_sort (cull == false; the cull-data pointers are unused) and xpr_bin_sort_cull.
static int32_t bin_sort_impl(bool cull, int64_t N, const float* depth, const int32_t* tile_rect,
                             const uint32_t* tile_count, const float* mean2d, const float* conic_opac, const float* lnv,
                             const float* lin_rec,
                             const xpr_camera* cam, const xpr_config* cfg, int64_t pair_capacity,
                             uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* tile_ranges,
                             int64_t* num_pairs_host, void* workspace, size_t workspace_bytes, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0 || pair_capacity < 0 || pair_capacity >= (1LL << 30)) return XPR_ERR_INVALID_ARG;
    if (N >= (1LL << 30)) return XPR_ERR_UNSUPPORTED;      // the look-back status words carry 30-bit counts
    // a batch of V views (xpr_config.views) is one image of V * tiles_y tile rows: view v owns rows [v tiles_y, (v+1) tiles_y)
    const int TW = tiles_x(cam), TH_view = tiles_y(cam), TH = TH_view * num_views(cfg);
    const int64_t T64 = (int64_t)TW * TH;
    if (T64 > (1 << 24) || TW > 0xffff) return XPR_ERR_UNSUPPORTED;   // row table: 16-bit columns
    const int32_t T = (int32_t)T64;
    const int STW = (TW + ST_EDGE - 1) >> ST_SHIFT, STH = (TH + ST_EDGE - 1) >> ST_SHIFT;
    const int32_t ST = STW * STH;
    if (!aligned(tile_ranges, 8) || !aligned(workspace, 256)) return XPR_ERR_INVALID_ARG;
    if (N > 0 && (!aligned(depth, 4) || !aligned(tile_rect, 16) || !aligned(tile_count, 4))) return XPR_ERR_INVALID_ARG;
    if (cull && N > 0 && (!aligned(mean2d, 8) || !aligned(conic_opac, 16) || !aligned(lnv, 4))) return XPR_ERR_INVALID_ARG;
    if (pair_capacity > 0 && (!aligned(keys_sorted, 8) || !aligned(vals_sorted, 4))) return XPR_ERR_INVALID_ARG;
    const Layout L = make_layout(N, pair_capacity, T);
    if (workspace_bytes < L.total) return XPR_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    Header* hdr = reinterpret_cast<Header*>(ws + L.header);
    const size_t scan_blocks = ((size_t)N + SCAN_ITEMS - 1) / SCAN_ITEMS;
    unsigned long long* compact_status = reinterpret_cast<unsigned long long*>(ws + L.scan_status);
    unsigned long long* scan_status = compact_status + scan_blocks + 1;
    uint32_t* vkey[2] = {reinterpret_cast<uint32_t*>(ws + L.vkey0), reinterpret_cast<uint32_t*>(ws + L.vkey1)};
    uint32_t* vidx[2] = {reinterpret_cast<uint32_t*>(ws + L.vidx0), reinterpret_cast<uint32_t*>(ws + L.vidx1)};
    uint32_t* status32 = reinterpret_cast<uint32_t*>(ws + L.status32);
    uint32_t* status64 = reinterpret_cast<uint32_t*>(ws + L.status64);
    uint32_t* final_status = reinterpret_cast<uint32_t*>(ws + L.final_status);
    int* tile_diff = reinterpret_cast<int*>(ws + L.tile_diff);
    uint32_t* seg_cnt = reinterpret_cast<uint32_t*>(ws + L.seg_cnt);
    uint32_t* seg_start = reinterpret_cast<uint32_t*>(ws + L.seg_start);
    uint32_t* chunk_start = reinterpret_cast<uint32_t*>(ws + L.chunk_start);
    // second pair buffer: the row table (4 bytes per row, rows < pair_capacity) in its first half, the sorted
    // supertile words (8 bytes each, at most pair_capacity / 2 of them) in its second half
    uint32_t* row_tab = reinterpret_cast<uint32_t*>(ws + L.keys_tmp);
    uint64_t* words_half = reinterpret_cast<uint64_t*>(ws + L.keys_tmp + align_up(4 * (size_t)pair_capacity, 256));
    const int l1_passes = digit_passes_for(ST);

    if (num_pairs_host) *num_pairs_host = 0;
    if (N == 0) {
        XPR_CUDA(cudaMemsetAsync(tile_ranges, 0, sizeof(uint32_t) * 2 * (size_t)T, st));
        XPR_CUDA(cudaMemsetAsync(ws + L.header, 0, sizeof(Header), st));       // pair count 0 for an asynchronous caller
        if (cfg->tile_order) {
            XPR_CUDA(launch_k(true, tile_order_kernel, dim3(1), dim3(1024), 0, st, tile_ranges, (uint32_t)T, cfg->tile_order));
            XPR_LAUNCH_CHECK();
        }
        return XPR_OK;
    }
    XPR_CUDA(cudaMemsetAsync(ws + L.header, 0, L.zero_end - L.header, st));   // header, chains, look-back words, counters
    // 1. visible Gaussians (index order) + depth-digit histograms
    XPR_CUDA(launch_k(true, compact_kernel, dim3((unsigned)scan_blocks), dim3(SCAN_THREADS), 0, st, N, depth, tile_count, hdr, compact_status, vkey[0],
                                                                   vidx[0]));
    XPR_LAUNCH_CHECK();
    // 2. the four depth digits, on the N_vis Gaussians (tiles counted for N; surplus tickets end the loop)
    const unsigned tiles32 = (unsigned)(((size_t)N + SORT_THREADS * IPT32 - 1) / (SORT_THREADS * IPT32));
    for (int p = 0; p < DEPTH_PASSES; ++p) {
        uint32_t* status = status32 + (size_t)p * RADIX * tiles32;
        const int a = p & 1, b = a ^ 1;
        // mantissa bytes: ~32 distinct digits per warp -> bitmap ranking; exponent byte: match.any
#define XPR_DEPTH_PASS(BITMAP_)                                                                          \
    launch_pass<uint32_t, IPT32, BITMAP_, 0>(tiles32, st, &hdr->n_vis, nullptr, 8 * p, p, vkey[a], vidx[a], \
                                             vkey[b], vidx[b], hdr, status)
        const cudaError_t e = (p < 3) ? XPR_DEPTH_PASS(true) : XPR_DEPTH_PASS(false);
#undef XPR_DEPTH_PASS
        XPR_CUDA(e);
    }   // DEPTH_PASSES is even: the list in rank order is back in vkey[0] / vidx[0]
    // 3. scans in rank order: rows and supertile words of the earlier Gaussians; every count stays on
    //    the device and later kernels read it there (persistent grids), so nothing waits for the host.
    //    vkey[1] / vidx[1] are free after the depth passes.
    uint32_t* row_base = vkey[1];
    uint32_t* l1_off = vidx[1];
    const int4* rect4 = reinterpret_cast<const int4*>(tile_rect);
    const unsigned sgrid = (unsigned)scan_blocks < 2u * PERSIST_CTAS ? (unsigned)scan_blocks : 2u * PERSIST_CTAS;
    XPR_CUDA(launch_k(true, rank_scan_kernel, dim3(sgrid), dim3(SCAN_THREADS), 0, st, vidx[0], rect4, tile_count, hdr, scan_status, row_base, l1_off,
                                                     (unsigned long long)pair_capacity));
    XPR_LAUNCH_CHECK();
    // 4. rows: surviving interval per (Gaussian, tile row) -> row table + difference array over the tile ids
    const unsigned rgrid = 148u * 16u;                               // grid-stride over the rows (count on the device)
    if (cull)
        XPR_CUDA(launch_k(true, rows_kernel<1>, dim3(rgrid), dim3(128), 0, st, TW, TH, TH_view, vidx[0], row_base, rect4, reinterpret_cast<const float2*>(mean2d),
                                              reinterpret_cast<const float4*>(conic_opac), lnv, nullptr, 0.0f, hdr, row_tab, tile_diff));
    else if (lin_rec && cfg->tile_cull != 0)
        XPR_CUDA(launch_k(true, rows_kernel<2>, dim3(rgrid), dim3(128), 0, st, TW, TH, TH_view, vidx[0], row_base, rect4, nullptr, nullptr, nullptr, lin_rec,
                                              (float)(-log(1.0 - (double)cfg->alpha_thresh)), hdr, row_tab, tile_diff));
    else
        XPR_CUDA(launch_k(true, rows_kernel<0>, dim3(rgrid), dim3(128), 0, st, TW, TH, TH_view, vidx[0], row_base, rect4, nullptr, nullptr, nullptr, nullptr, 0.0f,
                                              hdr, row_tab, tile_diff));
    XPR_LAUNCH_CHECK();
    // 5. supertile words in rank order; pass p of the supertile sort reads buffer p and writes buffer p + 1, the
    //    last one writes the half buffer (keys_sorted is free until the final pass)
    uint64_t* w0 = (l1_passes % 2 == 1) ? keys_sorted : words_half;
    uint64_t* w1 = (l1_passes % 2 == 1) ? words_half : keys_sorted;
    const unsigned egrid = (unsigned)(((size_t)N + 255) / 256) < 2u * 148u ? (unsigned)(((size_t)N + 255) / 256) : 2u * 148u;
#define XPR_EMIT(P_) XPR_CUDA(launch_k(false, l1_emit_kernel<P_>, dim3(egrid), dim3(256), 0, st, STW, (uint32_t)ST, vidx[0], rect4, l1_off, hdr, w0, seg_cnt))
    switch (l1_passes) {
        case 1: XPR_EMIT(1); break;
        case 2: XPR_EMIT(2); break;
        case 3: XPR_EMIT(3); break;
        default: XPR_EMIT(4); break;
    }
#undef XPR_EMIT
    XPR_LAUNCH_CHECK();
    // 6. per-tile counts and bases -> tile_ranges, I, capacity verdict; supertile segments and chunks
    XPR_CUDA(launch_k(true, tile_scan_kernel, dim3(1), dim3(TS_THREADS), 0, st, (uint32_t)T, (uint32_t)ST, (unsigned long long)pair_capacity, tile_diff, seg_cnt,
                                               reinterpret_cast<uint2*>(tile_ranges), seg_start, chunk_start, hdr));
    XPR_LAUNCH_CHECK();
    if (pair_capacity > 0) {
        // 7. stable sort of the words by supertile id (one pass per 8 bits)
        const unsigned tiles64 = (unsigned)(((size_t)pair_capacity / 2 + SORT_THREADS * IPT64 - 1) / (SORT_THREADS * IPT64)) + 1u;
        for (int p = 0; p < l1_passes; ++p) {
            uint32_t* status = status64 + (size_t)p * RADIX * tiles64;
            // pass 0: the words of one Gaussian are consecutive supertiles (distinct digits) -> bitmap ranking;
            // higher digits are nearly warp-uniform -> match.any
            const cudaError_t e = (p == 0)
                ? launch_pass<uint64_t, IPT64, true, 1>(tiles64, st, nullptr, &hdr->l1_eff, 32 + 8 * p, DEPTH_PASSES + p, w0,
                                                        nullptr, w1, nullptr, hdr, status)
                : launch_pass<uint64_t, IPT64, false, 1>(tiles64, st, nullptr, &hdr->l1_eff, 32 + 8 * p, DEPTH_PASSES + p, w0,
                                                         nullptr, w1, nullptr, hdr, status);
            XPR_CUDA(e);
            uint64_t* t = w0; w0 = w1; w1 = t;
        }   // the sorted words are in w0 == words_half
        // 8. the pairs, written once at their final position
        const size_t chunks_max = (size_t)pair_capacity / 2 / CHUNK + (size_t)ST + 1;
        const unsigned fgrid = chunks_max < (size_t)(148 * 8) ? (unsigned)chunks_max : 148u * 8u;
        XPR_CUDA(launch_k(true, final_kernel, dim3(fgrid), dim3(CHUNK), 0, st, TW, TH, STW, (uint32_t)ST, w0, seg_start, chunk_start, vkey[0], vidx[0], rect4,
                                             row_base, row_tab, reinterpret_cast<const uint2*>(tile_ranges), hdr,
                                             final_status, keys_sorted, vals_sorted));
        XPR_LAUNCH_CHECK();
    }
    if (cfg->tile_order) {                             // 9. scheduling order of the tiles for the compositing kernels
        XPR_CUDA(launch_k(true, tile_order_kernel, dim3(1), dim3(1024), 0, st, tile_ranges, (uint32_t)T, cfg->tile_order));
        XPR_LAUNCH_CHECK();
    }
    if (!num_pairs_host) return XPR_OK;                // asynchronous mode: the caller reads the count later
    unsigned long long counts[2] = {0, 0};             // I or the capacity that suffices; pairs in the output
    XPR_CUDA(cudaMemcpyAsync(counts, &hdr->total_pairs, sizeof(counts), cudaMemcpyDeviceToHost, st));
    XPR_CUDA(cudaStreamSynchronize(st));
    const unsigned long long total = counts[0];
    *num_pairs_host = ((int64_t)total > pair_capacity) ? (int64_t)total : (int64_t)counts[1];
    return ((int64_t)total > pair_capacity) ? XPR_ERR_CAPACITY : XPR_OK;
}

extern "C" int32_t xpr_bin_sort(int64_t N, const float* depth, const int32_t* tile_rect, const uint32_t* tile_count,
                                const xpr_camera* cam, const xpr_config* cfg, int64_t pair_capacity,
                                uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* tile_ranges,
                                int64_t* num_pairs_host, void* workspace, size_t workspace_bytes, void* stream) {
    if (cfg && cfg->tile_cull != 0) return XPR_ERR_INVALID_ARG;     // tile_cull needs the cull data: xpr_bin_sort_cull
    return bin_sort_impl(false, N, depth, tile_rect, tile_count, nullptr, nullptr, nullptr, nullptr, cam, cfg, pair_capacity,
                         keys_sorted, vals_sorted, tile_ranges, num_pairs_host, workspace, workspace_bytes, stream);
}

extern "C" int32_t xpr_bin_sort_cull(int64_t N, const float* depth, const int32_t* tile_rect,
                                     const uint32_t* tile_count, const float* mean2d, const float* conic_opac,
                                     const float* lnv, const xpr_camera* cam, const xpr_config* cfg,
                                     int64_t pair_capacity, uint64_t* keys_sorted, uint32_t* vals_sorted,
                                     uint32_t* tile_ranges, int64_t* num_pairs_host, void* workspace,
                                     size_t workspace_bytes, void* stream) {
    const bool cull = cfg && cfg->tile_cull != 0;
    return bin_sort_impl(cull, N, depth, tile_rect, tile_count, mean2d, conic_opac, lnv, nullptr, cam, cfg, pair_capacity,
                         keys_sorted, vals_sorted, tile_ranges, num_pairs_host, workspace, workspace_bytes, stream);
}

// xpr_bin_sort for XPR-LinPrim: the same binning and sort; with cfg->tile_cull != 0 the pairs are culled
// with the per-tile chord bound of Eq. 2 read from lin_rec[N,20] of xpr_lin_project.
extern "C" int32_t xpr_bin_sort_lin(int64_t N, const float* depth, const int32_t* tile_rect, const uint32_t* tile_count,
                                    const float* lin_rec, const xpr_camera* cam, const xpr_config* cfg,
                                    int64_t pair_capacity, uint64_t* keys_sorted, uint32_t* vals_sorted,
                                    uint32_t* tile_ranges, int64_t* num_pairs_host, void* workspace,
                                    size_t workspace_bytes, void* stream) {
    if (N > 0 && !aligned(lin_rec, 16)) return XPR_ERR_INVALID_ARG;
    if (cfg && num_views(cfg) != 1) return XPR_ERR_UNSUPPORTED;
    return bin_sort_impl(false, N, depth, tile_rect, tile_count, nullptr, nullptr, nullptr, lin_rec, cam, cfg, pair_capacity,
                         keys_sorted, vals_sorted, tile_ranges, num_pairs_host, workspace, workspace_bytes, stream);
}

// ---------------------------------------------------------------------------------------------
// xpr_bin_sort_static -- xpr_bin_sort / xpr_bin_sort_cull for callers that cannot allocate (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc): the workspace is a file-scope device array of
// XPR_STATIC_SCRATCH_BYTES that every GPU loading the library holds until the process exits.  The entry point calls no
// cudaMalloc / cudaFree / allocating library routine; inputs and outputs are still the caller's.
// In host code the array's NAME is a host-side stand-in, not a device address: its device address is taken once per
// device, with that device current, by cudaGetSymbolAddress (below) and that pointer is what the kernels get.
// All calls on a device share the array, which keeps the last call's contents: bin_sort_impl zero-fills everything
// that must start at zero (header, chains, look-back words, counters: bytes [header, zero_end)) at the start of EVERY
// call, and every other region is written before it is read.  Two calls that overlap on the GPU (different streams
// without an ordering between them) race on the array.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_xpr_static_scratch[XPR_STATIC_SCRATCH_BYTES];

static int32_t static_scratch_address(void** out) {
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static void* ptrs[MAX_DEV] = {};
    int dev = -1;
    XPR_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) return XPR_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptrs[dev]) {                      // set-up, once per device, with that device current
        void* p = nullptr;
        XPR_CUDA(cudaGetSymbolAddress(&p, g_xpr_static_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return XPR_ERR_UNSUPPORTED;
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return XPR_OK;
}

extern "C" int32_t xpr_bin_sort_static(int64_t N, const float* depth, const int32_t* tile_rect,
                                       const uint32_t* tile_count, const float* mean2d, const float* conic_opac,
                                       const float* lnv, const xpr_camera* cam, const xpr_config* cfg,
                                       int64_t pair_capacity, uint64_t* keys_sorted, uint32_t* vals_sorted,
                                       uint32_t* tile_ranges, int64_t* num_pairs_host, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0 || pair_capacity < 0 || pair_capacity >= (1LL << 30)) return XPR_ERR_INVALID_ARG;
    if (N >= (1LL << 30)) return XPR_ERR_UNSUPPORTED;
    const int64_t T64 = (int64_t)tiles_x(cam) * tiles_y(cam) * num_views(cfg);
    if (T64 > (1 << 24)) return XPR_ERR_UNSUPPORTED;
    // the sizes this entry point serves: those whose workspace fits the static array
    if (make_layout(N, pair_capacity, (int32_t)T64).total > (size_t)XPR_STATIC_SCRATCH_BYTES) return XPR_ERR_SCRATCH_LIMIT;
    void* ws = nullptr;
    if (int32_t s = static_scratch_address(&ws)) return s;
    const bool cull = cfg->tile_cull != 0;
    return bin_sort_impl(cull, N, depth, tile_rect, tile_count, mean2d, conic_opac, lnv, nullptr, cam, cfg, pair_capacity,
                         keys_sorted, vals_sorted, tile_ranges, num_pairs_host, ws, (size_t)XPR_STATIC_SCRATCH_BYTES, stream);
}
