// binsort.cu -- xpr_bin_sort / xpr_bin_sort_cull: tile binning and the hand-written device radix sort.
//
// Rasterizer stage of the paper: "prefix-sum of tile counts", "replicate",
// "assign tile id" x = x_min + (r mod w), y = y_min + floor(r / w), t = y W' + x, optional "cull"
// (tile_cull, Listing 1), "sort lexicographically by (tile id, depth)", "identify bounds".
// Key packing tile << 32 | depth bits is BASELINE.json:north_star (reading C10); ties keep ascending
// Gaussian index.
//
// The sort is one stable LSD radix sort of the 64-bit keys, 8 bits per pass, reorganised around three
// observations:
//  (1) the four low digits are the depth bits, which all pairs of a Gaussian share, and replication
//      preserves order.  So the four depth passes run on the visible Gaussians (N_vis keys) BEFORE
//      replication, pairs are emitted in that order, and only the tile-id digits (2 passes at 1080p)
//      run on the replicated pairs.
//  (2) once the Gaussians are in (depth, index) order, a pair only has to carry its tile id and the
//      RANK of its Gaussian in that order: the tile passes move 8-byte words (tile << 32 | rank), and
//      the last pass expands them to the 64-bit key (tile << 32 | depth bits) and the 32-bit value
//      (Gaussian index) through two rank-indexed tables.  The expansion happens while the words are
//      still in the INPUT order of that pass, where neighbouring lanes hold neighbouring ranks, so
//      the gathers are coalesced (a gather in output order costs one 32-byte sector per pair).
//  (3) the unit of replication is a ROW -- the run of consecutive tiles one Gaussian covers in one
//      tile row: pair r of a row is tile_start + r (no divmod), and tile_cull reduces to one
//      surviving interval per row (the kept tiles of a row are contiguous because the quadratic form
//      is convex), found with 3-4 evaluations of the exact per-tile predicate instead of one per tile;
//      pairs that fail tile_cull are never generated.
// The result is bit-identical to sorting the (key, value) pairs by all digits; HBM traffic per pair
// drops from 12 + 6*24 + 8 = 164 bytes to 8 + 16 + 20 = 44 bytes.  No count ever travels to the host
// inside the call (persistent grids sized for the capacity; optional read-back at the end).
//
// Kernels (all hand-written, no CUB):
//   compact_kernel   single-pass chained scan (decoupled look-back) of the visibility flags; writes
//                    (depth bits, index) of the visible Gaussians in index order + the 4 depth-digit
//                    histograms.
//   onesweep_kernel  one launch per 8-bit digit, least significant first: warp-striped loads,
//                    stable in-warp ranking (shared-memory bitmap or match.any), shared-memory digit
//                    counts, per-digit decoupled look-back across tiles, shared-memory staged scatter.
//                    Persistent CTAs draw tiles from a ticket counter.  Instantiated for 32-bit
//                    keys + values (Gaussians) and for 64-bit packed words (pairs).
//   scan_kernel<0>   chained scan of the row counts of the Gaussians in depth order -> row bases.
//   rows_kernel      one thread per row: first tile, rank, number of tiles (whole width, or with
//                    tile_cull the surviving interval settled by the per-tile predicate tile_keep).
//   scan_kernel<1>   chained scan of the pairs per row -> pair offsets, I, first row of every emit unit.
//   emit_kernel      pair-parallel, load-balanced replication: a unit is 2048 consecutive pairs
//                    whatever rows they belong to (row heads scattered into shared memory, max-scan,
//                    then one coalesced 8-byte store per pair) + the tile-digit histograms.
//   ranges_kernel    per-tile (start, end): one warp per tile, 32-ary search in the sorted keys.
#include "common.cuh"

namespace xpr {
namespace {

constexpr int RADIX_BITS = 8;
constexpr int RADIX = 1 << RADIX_BITS;
constexpr int DEPTH_PASSES = 4;             // 32 depth bits
constexpr int MAX_TILE_PASSES = 4;          // up to 2^31 tiles

constexpr int SCAN_THREADS = 256;           // compact / offsets: 8 warps x 256 items
constexpr int SCAN_WARPS = SCAN_THREADS / 32;
constexpr int SCAN_ROUNDS = 8;              // items per lane
constexpr int SCAN_ITEMS = SCAN_THREADS * SCAN_ROUNDS;
constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
static_assert(SORT_THREADS == RADIX, "one thread per digit");
constexpr int IPT32 = 4;                    // Gaussian-level passes: 1024 keys per tile (N_vis is small)
#ifndef XPR_IPT64
#define XPR_IPT64 16
#endif
constexpr int IPT64 = XPR_IPT64;            // pair-level passes: 4096 pairs per tile
constexpr int PERSIST_CTAS = 148 * 4;       // upper bound of the persistent grids
constexpr int EMIT_THREADS = 256, EMIT_PPT = 8, EMIT_PAIRS = EMIT_THREADS * EMIT_PPT;   // emit: 2048 pairs per unit
constexpr int EMIT_WARPS = EMIT_THREADS / 32;
constexpr int EMIT_SHIFT = 11;
static_assert(SCAN_ITEMS == EMIT_PAIRS, "unit_status is sized for one scan block per emit unit");
static_assert(EMIT_PAIRS == 1 << EMIT_SHIFT, "unit_first is indexed by pair offset >> EMIT_SHIFT");

constexpr uint32_t FLAG_PARTIAL = 1u << 30, FLAG_INCLUSIVE = 2u << 30, FLAG_MASK = 3u << 30, VALUE_MASK = ~FLAG_MASK;
constexpr unsigned long long SFLAG_PARTIAL = 1ull << 62, SFLAG_INCLUSIVE = 2ull << 62, SFLAG_MASK = 3ull << 62;

// Header at the start of the workspace (zeroed every call).
struct Header {
    unsigned long long total_pairs;          // I (first 8 bytes of the workspace: readable by the caller)
    unsigned long long pairs_out;            // pairs in the sorted output (second 8 bytes): total_pairs if it fits, else 0
    unsigned long long pairs_eff;            // what emit expands: total_pairs if pairs and rows fit pair_capacity, else 0
    unsigned long long rows_total;           // (Gaussian, tile row) segments of the visible Gaussians
    unsigned long long rows_eff;             // rows_total if it fits pair_capacity, else 0
    unsigned long long cand_total;           // candidate pairs: sum of tile_count (what pair_capacity must hold)
    uint32_t n_vis;                          // visible Gaussians
    uint32_t compact_ticket, rows_ticket, offsets_ticket, unit_ticket;
    uint32_t sort_ticket[DEPTH_PASSES + MAX_TILE_PASSES];
    uint32_t pad[5];
    uint32_t hist[(DEPTH_PASSES + MAX_TILE_PASSES) * RADIX];   // global digit histograms
};

struct Layout {
    size_t header, scan_status, vkey0, vidx0, vkey1, vidx1, status32, keys_tmp, status64, unit_status, unit_first, total;
};

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

inline int tile_passes_for(int32_t num_tiles) {   // at least one: the last pass also expands the packed words
    int bits = 0;
    while (bits < 31 && ((int64_t)1 << bits) < (int64_t)num_tiles) ++bits;
    const int p = (bits + RADIX_BITS - 1) / RADIX_BITS;
    return p < 1 ? 1 : p;
}

inline Layout make_layout(int64_t N, int64_t cap, int32_t num_tiles) {
    Layout L;
    size_t off = 0;
    const size_t n = (size_t)N, c = (size_t)cap;
    const size_t scan_blocks = (n + SCAN_ITEMS - 1) / SCAN_ITEMS;
    L.header = off; off = align_up(off + sizeof(Header), 256);
    L.scan_status = off; off = align_up(off + 8 * 2 * (scan_blocks + 1), 256);      // compact + offsets chains
    const size_t tiles32 = (n + SORT_THREADS * IPT32 - 1) / (SORT_THREADS * IPT32);
    L.status32 = off; off = align_up(off + 4 * (size_t)RADIX * tiles32 * DEPTH_PASSES, 256);
    const size_t tiles64 = (c + SORT_THREADS * IPT64 - 1) / (SORT_THREADS * IPT64);
    L.status64 = off; off = align_up(off + 4 * (size_t)RADIX * tiles64 * (size_t)tile_passes_for(num_tiles), 256);
    L.unit_status = off; off = align_up(off + 8 * (c / EMIT_PAIRS + 2), 256);    // emit's chain over units (tile_cull)
    // everything up to here is zeroed with one memset
    L.vkey0 = off; off = align_up(off + 4 * n, 256);
    L.vidx0 = off; off = align_up(off + 4 * n, 256);
    L.vkey1 = off; off = align_up(off + 4 * n, 256);
    L.vidx1 = off; off = align_up(off + 4 * n, 256);
    L.keys_tmp = off; off = align_up(off + 8 * c, 256);
    L.unit_first = off; off = align_up(off + 4 * (c / EMIT_PAIRS + 2), 256);   // one entry per EMIT_PAIRS pairs
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
__device__ __forceinline__ unsigned long long chain_lookback(uint32_t block, uint32_t btotal,
                                                             unsigned long long* __restrict__ status, int lane) {
    unsigned long long excl = 0;
    if (block == 0) {
        if (lane == 0) st_relaxed64(&status[0], SFLAG_INCLUSIVE | (unsigned long long)btotal);
        return 0;
    }
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
        const unsigned long long e = chain_lookback(block, btotal, status, lane);
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
// Chained scans in depth order ("prefix-sum of tile counts").  The unit of replication is
// a ROW: the run of consecutive tiles that one Gaussian covers in one tile row (all of its rectangle's
// row, or with tile_cull the surviving interval), because pair r of a row is simply tile_start + r.
//   MODE 0: values = tile rows h of the Gaussians in depth order -> row_base[rank], rows_total
//   MODE 1: values = pairs of the rows                          -> row_off[row] (+ one past the end),
//           unit_first[u] = the row that owns pair u * EMIT_PAIRS, total_pairs / pairs_out / pairs_eff
// ---------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(SCAN_THREADS)
scan_kernel(const uint32_t* __restrict__ vidx, const int4* __restrict__ rect, const uint32_t* __restrict__ tcount,
            Header* __restrict__ hdr, unsigned long long* __restrict__ status, uint32_t* out,
            uint32_t* __restrict__ aux /* MODE 1: unit_first */, uint32_t units_cap,
            unsigned long long pair_capacity) {
    __shared__ uint32_t s_warp[SCAN_WARPS];
    __shared__ uint32_t s_block;
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t n = (MODE == 0) ? hdr->n_vis : (uint32_t)hdr->rows_eff;
    uint32_t* const unit_first = aux;
    for (;;) {       // persistent: blocks of SCAN_ITEMS items are drawn from a ticket counter (= look-back order)
    __syncthreads();
    if (tid == 0) s_block = atomicAdd(MODE == 0 ? &hdr->rows_ticket : &hdr->offsets_ticket, 1u);
    __syncthreads();
    const uint32_t block = s_block;
    if ((uint64_t)block * SCAN_ITEMS >= n && block != 0) return;   // beyond the list: nobody waits on us
    const uint32_t s0 = block * (uint32_t)SCAN_ITEMS + (uint32_t)warp * (32 * SCAN_ROUNDS) + (uint32_t)lane;
    uint32_t val[SCAN_ROUNDS];
    unsigned long long cand = 0;                       // MODE 0: candidate pairs of this thread's Gaussians
#pragma unroll
    for (int r = 0; r < SCAN_ROUNDS; ++r) {
        const uint32_t s = s0 + r * 32;
        val[r] = 0u;
        if (s < n) {
            if (MODE == 0) {
                const uint32_t g = __ldg(vidx + s);
                const int4 q = __ldg(rect + g);
                val[r] = (uint32_t)(q.w - q.y);
                cand += __ldg(tcount + g);
            }
            else val[r] = out[s];                       // MODE 1 scans in place: counts in, offsets out
        }
    }
    uint32_t excl[SCAN_ROUNDS], wtotal = 0;
#pragma unroll
    for (int r = 0; r < SCAN_ROUNDS; ++r) {
        uint32_t incl = val[r];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        excl[r] = wtotal + incl - val[r];
        wtotal += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (MODE == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) cand += __shfl_xor_sync(0xffffffffu, cand, o);
        if (lane == 0 && cand) atomicAdd(&hdr->cand_total, cand);
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
        const unsigned long long e = chain_lookback(block, btotal, status, lane);
        if (lane == 0) s_base = e;
    }
    __syncthreads();
    const unsigned long long base = s_base;
    const bool last_block = (uint64_t)(block + 1) * SCAN_ITEMS >= n;
    const unsigned long long total = base + btotal;
#pragma unroll
    for (int r = 0; r < SCAN_ROUNDS; ++r) {
        const uint32_t s = s0 + r * 32;
        if (s < n) {
            const unsigned long long off = base + wbase + excl[r], end = off + val[r];
            out[s] = (uint32_t)off;
            if (MODE == 1) {
                // emit works in units of EMIT_PAIRS consecutive pairs: unit u starts inside this row's pairs
                // iff off <= EMIT_PAIRS u < end; then this row is the first one the unit needs
                for (unsigned long long u = (off + (EMIT_PAIRS - 1)) >> EMIT_SHIFT; (u << EMIT_SHIFT) < end && u < units_cap; ++u)
                    unit_first[u] = s;
            }
        }
    }
    if (tid == 0 && last_block) {
        if (MODE == 0) {
            hdr->rows_total = total;
            hdr->rows_eff = (total < pair_capacity) ? total : 0ull;    // over capacity: the row kernels do nothing
                                                                        // (strict: row_off has one entry past the rows)
        } else {
            out[n] = (uint32_t)total;                    // one past the end: a row's pairs are [row_off[s], row_off[s+1])
            // the capacity must hold the candidate pairs (sum of tile_count >= pairs, >= rows), as in xpr.h
            const unsigned long long rows = hdr->rows_total, cand = hdr->cand_total;
            const bool ok = cand <= pair_capacity && rows < pair_capacity;
            hdr->total_pairs = ok ? total : (cand > rows + 1 ? cand : rows + 1);
            hdr->pairs_out = ok ? total : 0ull;
            hdr->pairs_eff = ok ? total : 0ull;           // over capacity: the pair kernels do nothing
        }
    }
    if (last_block) return;
    }
}

__device__ __forceinline__ bool tile_keep(float mx, float my, float A, float B, float C, float lnv, uint32_t tx, uint32_t ty);

// ---------------------------------------------------------------------------------------------
// rows: one thread per visible Gaussian (in depth order) writes its h rows: first tile id, number of
// tiles, rank.  Without tile_cull a row is the whole width of the rectangle.  With tile_cull (PAPER
// L149 "Cull") it is the interval of tiles that pass tile_keep: the set {x : min_{y in row} q <= lnv}
// is an interval (q is convex), so the kernel estimates its two ends analytically (the ellipse
// {q = lnv} cut by the strip of the row: its extreme x, or its intersection with the strip's edges) and
// then settles each end with the exact per-tile predicate tile_keep -- the decision that defines the
// result (bit-identical to the oracle's) -- stepping while the predicate disagrees.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float approx_sqrt(float x) {   // the interval estimate needs no exact rounding
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <bool CULL>
__global__ void __launch_bounds__(128)
rows_kernel(int TW, const uint32_t* __restrict__ vidx, const uint32_t* __restrict__ row_base,
            const int4* __restrict__ rect, const float2* __restrict__ mean2d, const float4* __restrict__ conic_opac,
            const float* __restrict__ lnv, const Header* __restrict__ hdr, uint32_t* __restrict__ row_start,
            uint32_t* __restrict__ row_rank, uint32_t* __restrict__ row_cnt) {
    // one thread per row (grid-stride, a warp takes 32 consecutive rows).  The Gaussian of a row is the last one
    // whose first row is <= row: the warp finds it for its first row with a cooperative 32-ary search in the
    // strictly increasing row_base (4 dependent loads for 10^6 Gaussians instead of 20), loads the next 32 bases
    // with one coalesced read -- the 32 rows of the warp cannot span more Gaussians -- and every lane finishes
    // with a 5-step search over those through shuffles.
    const uint32_t n_rows = (uint32_t)hdr->rows_eff, n_vis = hdr->n_vis;
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
        row_rank[row] = s;
        const uint32_t g = vidx[s];
        const int4 r = rect[g];
        const int ty = r.y + (int)(row - row_base[s]);
        float mx = 0.f, my = 0.f, A = 0.f, B = 0.f, C = 0.f, L = 0.f, ext = 0.f, det = 0.f;
        if (CULL) {
            const float2 m = mean2d[g]; const float4 co = conic_opac[g];
            mx = m.x; my = m.y; A = co.x; B = co.y; C = co.z; L = lnv[g];
            det = A * C - B * B;
            ext = approx_sqrt(fmaxf(__fdividef(2.0f * L * C, det), 0.0f));   // half-width of the ellipse {q = L} in x
        }
        int xa = r.x, xb = r.z;                                 // kept tiles of this row: [xa, xb)
        if (CULL) {
            const auto keep = [&](int tx) { return tile_keep(mx, my, A, B, C, L, (uint32_t)tx, (uint32_t)ty); };
            // estimate: x extent of {q <= L} over dy in [lo, hi] (pixel-centre hull of the row)
            const float lo = (float)(TILE * ty) + 0.5f - my, hi = (float)(TILE * ty + TILE) - 0.5f - my;
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
            bool found = false;
            if (left <= right) {
                xa = max(r.x, min(r.z - 1, (int)floorf((mx + left - ((float)TILE - 0.5f)) * (1.0f / (float)TILE)) + 1));
                xb = max(xa, min(r.z - 1, (int)floorf((mx + right - 0.5f) * (1.0f / (float)TILE)))) + 1;   // exclusive
                // settle the left end with the exact predicate
                int t = xa;
                if (keep(t)) { while (t > r.x && keep(t - 1)) --t; found = true; }
                else { while (t < xb && !keep(t)) ++t; found = t < xb; }
                xa = t;
                if (found) {
                    t = max(xb - 1, xa);
                    if (keep(t)) { while (t + 1 < r.z && keep(t + 1)) ++t; }
                    else { while (t > xa && !keep(t)) --t; }
                    xb = t + 1;
                }
            }
            if (!found) {
                // the estimate saw nothing.  q_min over the row's tiles is convex in x, so if any tile is kept the
                // one nearest the row's minimiser x* is: x* = mx when the mean lies in the row's strip, else
                // mx - B c / A with c the strip edge nearest the mean.  Test it and its neighbours (rounding of
                // x*), then grow the interval with the predicate.
                const float c = (lo <= 0.0f && hi >= 0.0f) ? 0.0f : ((lo > 0.0f) ? lo : hi);
                const int tc = max(r.x, min(r.z - 1, (int)floorf((mx - B * c * rA) * (1.0f / (float)TILE))));
                int t = -1;
                if (keep(tc)) t = tc;
                else if (tc > r.x && keep(tc - 1)) t = tc - 1;
                else if (tc + 1 < r.z && keep(tc + 1)) t = tc + 1;
                if (t < 0) { xa = xb = r.x; }
                else {
                    xa = t; while (xa > r.x && keep(xa - 1)) --xa;
                    xb = t + 1; while (xb < r.z && keep(xb)) ++xb;
                }
            }
        }
        row_start[row] = (uint32_t)ty * (uint32_t)TW + (uint32_t)xa;
        row_cnt[row] = (uint32_t)(xb - xa);
    }
}

// ---------------------------------------------------------------------------------------------
// emit: replicate + assign tile id, pair-parallel and load-balanced.  A unit of work is
// EMIT_PAIRS consecutive pairs [p0, p1), whatever Gaussians they belong to (a near Gaussian covers
// thousands of tiles, and in depth order those come first):
//   1. warp 0 finds the Gaussian (in depth order) that owns pair p0 by a 32-ary search in voff;
//   2. the Gaussians that start inside [p0, p1) are loaded one per thread into shared memory
//      (offset, first tile id, rectangle width, 1/width) and their slot number is written at the
//      position of their first pair;
//   3. a max-scan over the positions gives every pair its slot;
//   4. pair j of a slot: r = j - offset, (ry, rx) = divmod(r, w), tile = tile0 + ry * TW + rx; one
//      coalesced 8-byte store of tile << 32 | rank; shared-memory histograms of the tile digits.
// CTAs are persistent (grid <= PERSIST_CTAS) so that the digit histograms are flushed to global
// memory once per CTA, not once per 2048 pairs.
// ---------------------------------------------------------------------------------------------
constexpr int EMIT_CAND = 2;                 // prefetched candidate Gaussians per thread and unit

// tile_cull of XPR-3DGS ("Cull", Listing 1, A.1.1 L435): true when the pair survives,
// i.e. unless min over the hull of the tile's pixel centres of 1/2 d^T K d exceeds lnv = ln(o / alpha_thresh)
// by more than the conservative margin.  Evaluation order and margin are reading C8 of DESIGN.md; every
// operation is individually rounded (explicit _rn intrinsics: this file is compiled with FMA contraction).
__device__ __forceinline__ bool tile_keep(float mx, float my, float A, float B, float C, float lnv, uint32_t tx, uint32_t ty) {
    const float ts = (float)TILE;
    const float x0 = __fadd_rn(__fmul_rn(ts, (float)tx), 0.5f), x1 = __fsub_rn(__fadd_rn(__fmul_rn(ts, (float)tx), ts), 0.5f);
    const float y0 = __fadd_rn(__fmul_rn(ts, (float)ty), 0.5f), y1 = __fsub_rn(__fadd_rn(__fmul_rn(ts, (float)ty), ts), 0.5f);
    const bool in_x = (mx >= x0) && (mx <= x1), in_y = (my >= y0) && (my <= y1);
    if (in_x && in_y) return true;
    const float margin = 1.0f / 262144.0f;   // 2^-18
    auto drop = [&](float dx, float dy) {
        const float a = __fmul_rn(__fmul_rn(__fmul_rn(0.5f, A), dx), dx), b = __fmul_rn(__fmul_rn(B, dx), dy),
                    c = __fmul_rn(__fmul_rn(__fmul_rn(0.5f, C), dy), dy);
        const float q = __fadd_rn(__fadd_rn(a, b), c);
        const float mag = __fadd_rn(__fadd_rn(__fadd_rn(fabsf(a), fabsf(b)), fabsf(c)), lnv);
        return q > __fadd_rn(lnv, __fmul_rn(mag, margin));
    };
    bool dropped = true;                      // dropped by every facing edge
    if (!in_x) {
        const float dx = __fsub_rn((mx < x0) ? x0 : x1, mx);
        float dy = __fdiv_rn(-__fmul_rn(B, dx), C);
        const float lo = __fsub_rn(y0, my), hi = __fsub_rn(y1, my);
        dy = (dy < lo) ? lo : dy; dy = (hi < dy) ? hi : dy;
        dropped = dropped && drop(dx, dy);
    }
    if (!in_y) {
        const float dy = __fsub_rn((my < y0) ? y0 : y1, my);
        float dx = __fdiv_rn(-__fmul_rn(B, dy), A);
        const float lo = __fsub_rn(x0, mx), hi = __fsub_rn(x1, mx);
        dx = (dx < lo) ? lo : dx; dx = (hi < dx) ? hi : dx;
        dropped = dropped && drop(dx, dy);
    }
    return !dropped;
}

template <int TILE_PASSES>
__global__ void __launch_bounds__(EMIT_THREADS)
emit_kernel(const uint32_t* __restrict__ row_off, const uint32_t* __restrict__ row_start,
            const uint32_t* __restrict__ row_rank, const uint32_t* __restrict__ unit_first, Header* __restrict__ hdr,
            uint64_t* __restrict__ words) {
    __shared__ uint4 s_slot[EMIT_PAIRS];             // pair offset of the row, its first tile id, rank of its Gaussian, -
    __shared__ __align__(16) uint16_t s_mark[EMIT_PAIRS];
    __shared__ uint32_t s_hist[MAX_TILE_PASSES * RADIX];
    __shared__ uint32_t s_wmax[EMIT_WARPS];
    __shared__ uint32_t s_unit[2];                   // tickets: this unit's successor (double buffered)
    constexpr int tile_passes = TILE_PASSES;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t n_rows = (uint32_t)hdr->rows_eff;
    const uint32_t I = (uint32_t)hdr->pairs_eff;
    const uint32_t units = (I + EMIT_PAIRS - 1) / EMIT_PAIRS;
    for (int b = tid; b < tile_passes * RADIX; b += EMIT_THREADS) s_hist[b] = 0u;
    // units are drawn from a ticket counter; the first row of every unit was recorded by the offsets scan
    // (unit_first), so a unit needs no search; the candidate rows of the CTA's NEXT unit are prefetched into
    // registers while the current one is expanded (the dependent loads are off the critical path)
    uint32_t c_off[EMIT_CAND], c_end[EMIT_CAND], c_start[EMIT_CAND], c_rank[EMIT_CAND];
    auto load_candidates = [&](uint32_t first) {
#pragma unroll
        for (int c = 0; c < EMIT_CAND; ++c) {
            const uint32_t s = first + (uint32_t)c * EMIT_THREADS + (uint32_t)tid;
            c_off[c] = 0xffffffffu; c_end[c] = 0xffffffffu;  // beyond the list: never < a pair index
            if (s < n_rows) { c_off[c] = row_off[s]; c_end[c] = row_off[s + 1]; c_start[c] = row_start[s]; c_rank[c] = row_rank[s]; }
        }
    };
    if (tid == 0) s_unit[0] = atomicAdd(&hdr->unit_ticket, 1u);
    __syncthreads();
    uint32_t unit = s_unit[0], first = 0, next_first = 0;
    if (unit < units) { first = unit_first[unit]; load_candidates(first); }

    for (int phase = 0; unit < units; phase ^= 1) {
        const uint32_t p0 = unit * (uint32_t)EMIT_PAIRS, p1 = min(I, p0 + (uint32_t)EMIT_PAIRS);
        if (tid == 0) s_unit[phase ^ 1] = atomicAdd(&hdr->unit_ticket, 1u);      // the unit after this one
        __syncthreads();                              // previous unit done with the shared arrays
        reinterpret_cast<uint4*>(s_mark)[tid] = make_uint4(0u, 0u, 0u, 0u);      // 8 marks per thread
        // rows first .. cover [p0, p1); at most EMIT_PAIRS of them are non-empty (each owns a pair of the
        // unit), empty rows (tile_cull) own nothing and are skipped
        const int overflow = __syncthreads_or(c_off[EMIT_CAND - 1] < p1 && tid == EMIT_THREADS - 1);
        const uint32_t next_unit = s_unit[phase ^ 1];
        const bool has_next = next_unit < units;
        if (has_next) next_first = unit_first[next_unit];
#pragma unroll
        for (int c = 0; c < EMIT_CAND; ++c) {
            if (c_off[c] < p1 && c_end[c] > c_off[c]) {
                const uint32_t pos = c_off[c] > p0 ? c_off[c] - p0 : 0u;    // distinct for distinct non-empty rows
                s_slot[pos] = make_uint4(c_off[c], c_start[c], c_rank[c], 0u);
                s_mark[pos] = (uint16_t)pos;
            }
        }
        if (overflow) {
            // more rows start in this unit than were prefetched (tiny Gaussians): load the rest now
            for (uint32_t k = (uint32_t)(EMIT_CAND * EMIT_THREADS) + tid;; k += EMIT_THREADS) {
                const uint32_t s = first + k;
                if (s >= n_rows) break;
                const uint32_t off = row_off[s];
                if (off >= p1) break;
                if (row_off[s + 1] > off) {
                    s_slot[off - p0] = make_uint4(off, row_start[s], row_rank[s], 0u);
                    s_mark[off - p0] = (uint16_t)(off - p0);
                }
            }
        }
        if (has_next) { first = next_first; load_candidates(first); }   // consumed in the next iteration
        __syncthreads();
        {   // inclusive max-scan of the marks (thread t owns positions 8t .. 8t+7): slot of every pair
            uint4 mv = reinterpret_cast<uint4*>(s_mark)[tid];
            uint32_t m[8] = {mv.x & 0xffffu, mv.x >> 16, mv.y & 0xffffu, mv.y >> 16,
                             mv.z & 0xffffu, mv.z >> 16, mv.w & 0xffffu, mv.w >> 16};
#pragma unroll
            for (int q = 1; q < 8; ++q) m[q] = max(m[q], m[q - 1]);
            uint32_t incl = m[7];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) incl = max(incl, __shfl_up_sync(0xffffffffu, incl, o));
            if (lane == 31) s_wmax[warp] = incl;
            uint32_t excl = __shfl_up_sync(0xffffffffu, incl, 1);
            if (lane == 0) excl = 0u;
            __syncthreads();
#pragma unroll
            for (int w = 0; w < EMIT_WARPS; ++w)
                if (w < warp) excl = max(excl, s_wmax[w]);
#pragma unroll
            for (int q = 0; q < 8; ++q) m[q] = max(m[q], excl);
            reinterpret_cast<uint4*>(s_mark)[tid] = make_uint4(m[0] | (m[1] << 16), m[2] | (m[3] << 16),
                                                               m[4] | (m[5] << 16), m[6] | (m[7] << 16));
        }
        __syncthreads();
        // pair j belongs to the row whose first pair is the nearest mark at or before it: tile = first tile of
        // the row + (j - offset of the row).  The loads of the 8 pairs of a thread are issued together.
        uint32_t kk[EMIT_PPT];
        uint4 sl[EMIT_PPT];
#pragma unroll
        for (int it = 0; it < EMIT_PPT; ++it) kk[it] = s_mark[min((uint32_t)it * EMIT_THREADS + (uint32_t)tid, p1 - p0 - 1u)];
#pragma unroll
        for (int it = 0; it < EMIT_PPT; ++it) sl[it] = s_slot[kk[it]];
#pragma unroll
        for (int it = 0; it < EMIT_PPT; ++it) {
            const uint32_t j = p0 + (uint32_t)it * EMIT_THREADS + (uint32_t)tid;
            const bool valid = j < p1;                 // false only in the tail of the last unit
            const uint32_t tile = sl[it].y + (j - sl[it].x);
            if (valid) {
                words[j] = ((uint64_t)tile << 32) | (uint64_t)sl[it].z;
                atomicAdd(&s_hist[tile & 255u], 1u);   // consecutive tiles -> distinct banks
            }
            // higher tile digits are nearly warp-uniform: aggregate with match.any before the atomic
#pragma unroll
            for (int d = 1; d < tile_passes; ++d) {
                const uint32_t dig = valid ? ((tile >> (8 * d)) & 255u) : 0xffffffffu;
                const uint32_t peers = __match_any_sync(0xffffffffu, dig);
                if (valid && (peers & ((1u << lane) - 1u)) == 0u) atomicAdd(&s_hist[d * RADIX + dig], (uint32_t)__popc(peers));
            }
        }
        unit = next_unit;
    }
    __syncthreads();
    for (int b = tid; b < tile_passes * RADIX; b += EMIT_THREADS) {
        const uint32_t v = s_hist[b];
        if (v) atomicAdd(&hdr->hist[DEPTH_PASSES * RADIX + b], v);
    }
}

// ---------------------------------------------------------------------------------------------
// onesweep digit pass.  MODE 0: 32-bit keys + 32-bit values (the depth passes on Gaussians);
// MODE 1: 64-bit packed words tile << 32 | rank, no value; MODE 2: the last tile pass: reads words and,
// when staging them in shared memory, expands each to key = tile << 32 | tab_key[rank], value = tab_val[rank].
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

#ifndef XPR_P2_BITMAP
#define XPR_P2_BITMAP 1
#endif
#ifndef XPR_P1_BITMAP
#define XPR_P1_BITMAP 1
#endif
#ifndef XPR_SORT_MINB64
#define XPR_SORT_MINB64 4
#endif
template <class KeyT, int IPT, bool BITMAP, int MODE>
#ifndef XPR_SORT_MINB_M2
#define XPR_SORT_MINB_M2 3
#endif
__global__ void __launch_bounds__(SORT_THREADS, MODE == 2 ? XPR_SORT_MINB_M2 : (sizeof(KeyT) == 8 ? XPR_SORT_MINB64 : 4))   // MODE 2: 66 KB of shared memory
onesweep_kernel(const uint32_t* __restrict__ n_dev32, const unsigned long long* __restrict__ n_dev64, int shift,
                int hist_row, int ticket_row, const KeyT* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                KeyT* __restrict__ keys_out, uint32_t* __restrict__ vals_out, Header* __restrict__ hdr,
                uint32_t* __restrict__ status /* [tiles][RADIX] of this pass */,
                const uint32_t* __restrict__ tab_key, const uint32_t* __restrict__ tab_val) {
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
            if constexpr (MODE == 2) {
                const uint32_t loc = wofs + (uint32_t)it * 32u;
                const uint32_t r = (loc < tile_n) ? (uint32_t)key[it] : 0u;     // rank; 0 for the padding
                S.keys[pos] = (key[it] & ~(KeyT)0xffffffffu) | (KeyT)__ldg(tab_key + r);
                S.vals[pos] = __ldg(tab_val + r);
            } else {
                S.keys[pos] = key[it];
                if constexpr (HAS_VAL) {
                    const uint32_t loc = wofs + (uint32_t)it * 32u;
                    S.vals[pos] = (loc < tile_n) ? vals_in[tile_base + loc] : 0u;
                }
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
// per-tile bounds ("records each segment's start b_j and count c_j"): one warp per tile
// finds the first sorted key of tile t and of tile t+1 by a 32-ary search; an empty tile gets (0, 0).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t warp_lower_bound_tile(const uint64_t* __restrict__ keys, uint32_t n, uint32_t t,
                                                          int lane) {
    uint32_t lo = 0, hi = n;                   // answer in [lo, hi]; hi == n or tile(keys[hi]) >= t
    while (hi > lo) {
        const uint32_t len = hi - lo, stride = (len + 31u) / 32u;
        const uint32_t probe = min(lo + ((uint32_t)lane + 1u) * stride - 1u, hi - 1u);
        const uint32_t b = __ballot_sync(0xffffffffu, (uint32_t)(keys[probe] >> 32) >= t);
        if (b == 0u) { lo = hi; break; }
        const uint32_t f = (uint32_t)__ffs(b) - 1u;
        hi = min(lo + (f + 1u) * stride - 1u, hi - 1u);
        lo = lo + f * stride;
    }
    return lo;
}

__global__ void __launch_bounds__(256)
ranges_kernel(const unsigned long long* __restrict__ pairs_out, uint32_t T, const uint64_t* __restrict__ keys,
              uint32_t* __restrict__ ranges) {
    const uint32_t I = (uint32_t)*pairs_out;
    const uint32_t t = blockIdx.x * 8u + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (t >= T) return;
    const uint32_t b = warp_lower_bound_tile(keys, I, t, lane);
    const uint32_t e = warp_lower_bound_tile(keys, I, t + 1u, lane);
    if (lane == 0) reinterpret_cast<uint2*>(ranges)[t] = (e > b) ? make_uint2(b, e) : make_uint2(0u, 0u);
}

// pair_capacity == 0 (a caller probing for the size): the row / pair kernels do not run, so the capacity the call
// needs -- the candidate pairs, and one more than the rows -- is put where scan_kernel<1> would have put it.
__global__ void capacity_probe_kernel(Header* __restrict__ hdr) {
    const unsigned long long rows = hdr->rows_total, cand = hdr->cand_total;
    hdr->total_pairs = (cand > rows + 1) ? cand : ((rows > 0 || cand > 0) ? rows + 1 : 0ull);
    hdr->pairs_out = 0ull;
    hdr->pairs_eff = 0ull;
}

// Scheduling aid for the compositing kernels (xpr_config.tile_order): the tile indices by decreasing list length,
// in 1024 length classes (counting sort, one CTA: T is a few thousand).  Heaviest tiles first means the last wave
// of a compositing launch is made of short tiles.
__global__ void __launch_bounds__(1024)
tile_order_kernel(const uint32_t* __restrict__ ranges, uint32_t T, uint32_t* __restrict__ order) {
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
    *bytes = make_layout(N, pair_capacity, num_tiles).total;
    return XPR_OK;
}

template <class KeyT, int IPT, bool BITMAP, int MODE>
static cudaError_t launch_pass(unsigned tiles, cudaStream_t st, const uint32_t* n32, const unsigned long long* n64,
                               int shift, int row, const KeyT* kin, const uint32_t* vin, KeyT* kout, uint32_t* vout,
                               Header* hdr, uint32_t* status, const uint32_t* tab_key, const uint32_t* tab_val) {
    const size_t smem = sizeof(SortSmem<KeyT, IPT, MODE != 1>);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(onesweep_kernel<KeyT, IPT, BITMAP, MODE>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const unsigned grid = tiles < (unsigned)PERSIST_CTAS ? tiles : (unsigned)PERSIST_CTAS;
    onesweep_kernel<KeyT, IPT, BITMAP, MODE><<<grid, SORT_THREADS, smem, st>>>(n32, n64, shift, row, row, kin, vin, kout,
                                                                              vout, hdr, status, tab_key, tab_val);
    return cudaGetLastError();
}

// Common body of xpr_bin_sort (cull == false; the cull-data pointers are unused) and xpr_bin_sort_cull.
static int32_t bin_sort_impl(bool cull, int64_t N, const float* depth, const int32_t* tile_rect,
                             const uint32_t* tile_count, const float* mean2d, const float* conic_opac, const float* lnv,
                             const xpr_camera* cam, const xpr_config* cfg, int64_t pair_capacity,
                             uint64_t* keys_sorted, uint32_t* vals_sorted, uint32_t* tile_ranges,
                             int64_t* num_pairs_host, void* workspace, size_t workspace_bytes, void* stream) {
    if (int32_t s = check_cam_cfg(cam, cfg)) return s;
    if (N < 0 || pair_capacity < 0 || pair_capacity >= (1LL << 30)) return XPR_ERR_INVALID_ARG;
    if (N >= (1LL << 30)) return XPR_ERR_UNSUPPORTED;      // the look-back status words carry 30-bit counts
    const int TW = tiles_x(cam), TH = tiles_y(cam);
    const int64_t T64 = (int64_t)TW * TH;
    if (T64 > 0x7fffffffLL) return XPR_ERR_UNSUPPORTED;
    const int32_t T = (int32_t)T64;
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
    unsigned long long* offsets_status = compact_status + scan_blocks + 1;
    uint32_t* vkey[2] = {reinterpret_cast<uint32_t*>(ws + L.vkey0), reinterpret_cast<uint32_t*>(ws + L.vkey1)};
    uint32_t* vidx[2] = {reinterpret_cast<uint32_t*>(ws + L.vidx0), reinterpret_cast<uint32_t*>(ws + L.vidx1)};
    uint32_t* status32 = reinterpret_cast<uint32_t*>(ws + L.status32);
    uint64_t* keys_tmp = reinterpret_cast<uint64_t*>(ws + L.keys_tmp);
    uint32_t* status64 = reinterpret_cast<uint32_t*>(ws + L.status64);
    const int tpasses = tile_passes_for(T);

    if (num_pairs_host) *num_pairs_host = 0;
    if (N == 0) {
        XPR_CUDA(cudaMemsetAsync(tile_ranges, 0, sizeof(uint32_t) * 2 * (size_t)T, st));
        XPR_CUDA(cudaMemsetAsync(ws + L.header, 0, sizeof(Header), st));       // pair count 0 for an asynchronous caller
        if (cfg->tile_order) {
            tile_order_kernel<<<1, 1024, 0, st>>>(tile_ranges, (uint32_t)T, cfg->tile_order);
            XPR_LAUNCH_CHECK();
        }
        return XPR_OK;
    }
    XPR_CUDA(cudaMemsetAsync(ws + L.header, 0, L.vkey0 - L.header, st));   // header, scan chains, look-back status words
    // 1. visible Gaussians (index order) + depth-digit histograms
    compact_kernel<<<(unsigned)scan_blocks, SCAN_THREADS, 0, st>>>(N, depth, tile_count, hdr, compact_status, vkey[0],
                                                                   vidx[0]);
    XPR_LAUNCH_CHECK();
    // 2. the four depth digits, on the N_vis Gaussians (tiles counted for N; surplus tickets end the loop)
    const unsigned tiles32 = (unsigned)(((size_t)N + SORT_THREADS * IPT32 - 1) / (SORT_THREADS * IPT32));
    for (int p = 0; p < DEPTH_PASSES; ++p) {
        uint32_t* status = status32 + (size_t)p * RADIX * tiles32;
        const int a = p & 1, b = a ^ 1;
        // mantissa bytes: ~32 distinct digits per warp -> bitmap ranking; exponent byte: ballots
#define XPR_DEPTH_PASS(BITMAP_)                                                                          \
    launch_pass<uint32_t, IPT32, BITMAP_, 0>(tiles32, st, &hdr->n_vis, nullptr, 8 * p, p, vkey[a], vidx[a], \
                                             vkey[b], vidx[b], hdr, status, nullptr, nullptr)
        const cudaError_t e = (p < 3) ? XPR_DEPTH_PASS(true) : XPR_DEPTH_PASS(false);
#undef XPR_DEPTH_PASS
        XPR_CUDA(e);
    }   // DEPTH_PASSES is even: the sorted list is back in vkey[0] / vidx[0]
    // 3. rows: a row is the run of consecutive tiles one Gaussian covers in one tile row;
    //    scan of the row counts in depth order, the row table (with tile_cull: the surviving interval), scan
    //    of the pairs per row.  Every count stays on the device: later kernels read it there (grids are sized
    //    for pair_capacity), so nothing waits for the host.
    //    Scratch: the word buffer emission does not write to (free until pass 1) holds first tile + rank of
    //    the rows, vals_sorted (free until the last pass) their pair offsets, vkey[1]/vidx[1] (free after the
    //    depth passes) row bases and counts... all bounded by rows <= candidate pairs <= pair_capacity.
    uint64_t* w0 = (tpasses % 2 == 0) ? keys_sorted : keys_tmp;
    uint64_t* w1 = (tpasses % 2 == 0) ? keys_tmp : keys_sorted;
    uint32_t* row_base = vkey[1];
    uint32_t* unit_first = reinterpret_cast<uint32_t*>(ws + L.unit_first);
    unsigned long long* unit_status = reinterpret_cast<unsigned long long*>(ws + L.unit_status);
    const unsigned units_cap = (unsigned)((pair_capacity + EMIT_PAIRS - 1) / EMIT_PAIRS);
    const unsigned tiles64 = (unsigned)((pair_capacity + SORT_THREADS * IPT64 - 1) / (SORT_THREADS * IPT64));
    const int4* rect4 = reinterpret_cast<const int4*>(tile_rect);
    uint32_t* row_start = reinterpret_cast<uint32_t*>(w1);          // [pair_capacity]
    uint32_t* row_rank = row_start + pair_capacity;                  // [pair_capacity]
    const unsigned sgrid0 = (unsigned)scan_blocks < 2u * PERSIST_CTAS ? (unsigned)scan_blocks : 2u * PERSIST_CTAS;
    scan_kernel<0><<<sgrid0, SCAN_THREADS, 0, st>>>(vidx[0], rect4, tile_count, hdr, offsets_status, row_base, nullptr, 0u,
                                                    (unsigned long long)pair_capacity);
    XPR_LAUNCH_CHECK();
    if (pair_capacity > 0) {
        uint32_t* row_off = vals_sorted;                                 // counts, scanned in place; [rows + 1], rows < pair_capacity
        const unsigned rgrid = 148u * 16u;                               // grid-stride over the rows (count on the device)
        if (cull)
            rows_kernel<true><<<rgrid, 128, 0, st>>>(TW, vidx[0], row_base, rect4, reinterpret_cast<const float2*>(mean2d),
                                                     reinterpret_cast<const float4*>(conic_opac), lnv, hdr, row_start,
                                                     row_rank, row_off);
        else
            rows_kernel<false><<<rgrid, 128, 0, st>>>(TW, vidx[0], row_base, rect4, nullptr, nullptr, nullptr, hdr,
                                                      row_start, row_rank, row_off);
        XPR_LAUNCH_CHECK();
        const unsigned oblocks = (unsigned)(((size_t)pair_capacity + SCAN_ITEMS - 1) / SCAN_ITEMS);
        const unsigned sgrid1 = oblocks < 2u * PERSIST_CTAS ? oblocks : 2u * PERSIST_CTAS;
        scan_kernel<1><<<sgrid1, SCAN_THREADS, 0, st>>>(nullptr, nullptr, nullptr, hdr, unit_status, row_off, unit_first,
                                                        units_cap + 1u, (unsigned long long)pair_capacity);
        XPR_LAUNCH_CHECK();
        // 4. replicate in depth order as packed words; pass p reads buffer p and writes buffer p+1, the last
        //    one writes keys_sorted / vals_sorted, so emission starts in keys_sorted when tpasses is even
        const unsigned egrid = units_cap < (unsigned)PERSIST_CTAS ? units_cap : (unsigned)PERSIST_CTAS;
#define XPR_EMIT(TP) emit_kernel<TP><<<egrid, EMIT_THREADS, 0, st>>>(row_off, row_start, row_rank, unit_first, hdr, w0)
        switch (tpasses) {
            case 1: XPR_EMIT(1); break;
            case 2: XPR_EMIT(2); break;
            case 3: XPR_EMIT(3); break;
            default: XPR_EMIT(4); break;
        }
#undef XPR_EMIT
        XPR_LAUNCH_CHECK();
        // 5. the tile-id digits, on the I pairs
        for (int p = 0; p < tpasses; ++p) {
            uint32_t* status = status64 + (size_t)p * RADIX * tiles64;
            const int row = DEPTH_PASSES + p, shift = 32 + 8 * p;
            const bool last = (p == tpasses - 1);
            // bitmap ranking: consecutive pairs of a Gaussian are consecutive tiles (digit 0); after pass 1 a
            // warp holds many distinct high digits.  MODE 1: words -> words; MODE 2 (last pass): expand to key + value
#define XPR_TILE_PASS(BITMAP_, MODE_, VOUT_, TK_, TV_)                                                    \
    launch_pass<uint64_t, IPT64, BITMAP_, MODE_>(tiles64, st, nullptr, &hdr->pairs_out, shift, row, w0, nullptr, \
                                                 w1, VOUT_, hdr, status, TK_, TV_)
            const bool bitmap = (p == 0 && XPR_P1_BITMAP) || (p > 0 && XPR_P2_BITMAP);
            cudaError_t e;
            if (!last) e = bitmap ? XPR_TILE_PASS(true, 1, nullptr, nullptr, nullptr)
                                  : XPR_TILE_PASS(false, 1, nullptr, nullptr, nullptr);
            else       e = bitmap ? XPR_TILE_PASS(true, 2, vals_sorted, vkey[0], vidx[0])
                                  : XPR_TILE_PASS(false, 2, vals_sorted, vkey[0], vidx[0]);
#undef XPR_TILE_PASS
            XPR_CUDA(e);
            uint64_t* t = w0; w0 = w1; w1 = t;
        }
    } else {
        capacity_probe_kernel<<<1, 1, 0, st>>>(hdr);       // visible Gaussians but no room at all: XPR_ERR_CAPACITY below
        XPR_LAUNCH_CHECK();
    }
    // 6. per-tile ranges ((0, 0) for every tile when there are no pairs or they exceed the capacity)
    ranges_kernel<<<((unsigned)T + 7) / 8, 256, 0, st>>>(&hdr->pairs_out, (uint32_t)T, keys_sorted, tile_ranges);
    XPR_LAUNCH_CHECK();
    if (cfg->tile_order) {                             // 7. scheduling order of the tiles for the compositing kernels
        tile_order_kernel<<<1, 1024, 0, st>>>(tile_ranges, (uint32_t)T, cfg->tile_order);
        XPR_LAUNCH_CHECK();
    }
    if (!num_pairs_host) return XPR_OK;                // asynchronous mode: the caller reads the count later
    unsigned long long counts[2] = {0, 0};             // candidates I (must fit the capacity), pairs in the output
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
    return bin_sort_impl(false, N, depth, tile_rect, tile_count, nullptr, nullptr, nullptr, cam, cfg, pair_capacity,
                         keys_sorted, vals_sorted, tile_ranges, num_pairs_host, workspace, workspace_bytes, stream);
}

extern "C" int32_t xpr_bin_sort_cull(int64_t N, const float* depth, const int32_t* tile_rect,
                                     const uint32_t* tile_count, const float* mean2d, const float* conic_opac,
                                     const float* lnv, const xpr_camera* cam, const xpr_config* cfg,
                                     int64_t pair_capacity, uint64_t* keys_sorted, uint32_t* vals_sorted,
                                     uint32_t* tile_ranges, int64_t* num_pairs_host, void* workspace,
                                     size_t workspace_bytes, void* stream) {
    const bool cull = cfg && cfg->tile_cull != 0;
    return bin_sort_impl(cull, N, depth, tile_rect, tile_count, mean2d, conic_opac, lnv, cam, cfg, pair_capacity,
                         keys_sorted, vals_sorted, tile_ranges, num_pairs_host, workspace, workspace_bytes, stream);
}
