// binsort.cu -- xpr_bin_sort: tile binning and the hand-written device radix sort.
//
// Rasterizer stage of the paper: "prefix-sum of tile counts", "replicate",
// "assign tile id" x = x_min + (r mod w), y = y_min + floor(r / w), t = y W' + x, "sort
// lexicographically by (tile id, depth)", "identify bounds".  Key packing tile << 32 | depth bits
// is BASELINE.json:north_star (reading C10); ties keep ascending Gaussian index (stable sort on
// index-ordered emission).
//
// Kernels (all hand-written, no CUB):
//   emit_kernel      fused single-pass chained scan (decoupled look-back over 256-Gaussian blocks)
//                    + load-balanced pair emission (coalesced 8-byte key / 4-byte value stores)
//                    + all radix digit histograms (per-Gaussian for the depth digits, per-pair for
//                    the tile digits), so the sort never re-reads the keys to histogram them.
//   onesweep_kernel  one launch per 8-bit digit, least significant first: warp-striped loads,
//                    stable in-warp ranking with match.any, shared-memory digit counts, per-digit
//                    decoupled look-back across CTAs, shared-memory staged scatter.
//   ranges_kernel    per-tile (start, end) from the sorted keys.
#include "common.cuh"

namespace xpr {
namespace {

constexpr int RADIX_BITS = 8;
constexpr int RADIX = 1 << RADIX_BITS;
constexpr int MAX_PASSES = 8;

constexpr int EMIT_THREADS = 256;           // Gaussians per emit block (one per thread)

constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_IPT = 16;                // keys per thread
constexpr int SORT_TILE = SORT_THREADS * SORT_IPT;   // 4096 pairs per CTA
static_assert(SORT_THREADS == RADIX, "one thread per digit");

constexpr uint32_t FLAG_PARTIAL = 1u << 30, FLAG_INCLUSIVE = 2u << 30, FLAG_MASK = 3u << 30, VALUE_MASK = ~FLAG_MASK;
constexpr unsigned long long SFLAG_PARTIAL = 1ull << 62, SFLAG_INCLUSIVE = 2ull << 62, SFLAG_MASK = 3ull << 62;

// Header at the start of the workspace (zeroed every call).
struct Header {
    unsigned long long total_pairs;          // I
    uint32_t emit_ticket;
    uint32_t sort_ticket[MAX_PASSES];
    uint32_t pad[7];
    uint32_t hist[MAX_PASSES * RADIX];       // global digit histograms
};

struct Layout {
    size_t header, scan_status, keys_tmp, vals_tmp, sort_status, total;
};

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

inline int num_passes_for(int32_t num_tiles) {
    int bits = 0;
    while (bits < 32 && ((int64_t)1 << bits) < (int64_t)num_tiles) ++bits;
    return (32 + bits + RADIX_BITS - 1) / RADIX_BITS;
}

inline Layout make_layout(int64_t N, int64_t cap, int32_t num_tiles) {
    Layout L;
    size_t off = 0;
    L.header = off; off = align_up(off + sizeof(Header), 256);
    const size_t emit_blocks = (size_t)((N + EMIT_THREADS - 1) / EMIT_THREADS);
    L.scan_status = off; off = align_up(off + 8 * (emit_blocks + 1), 256);
    L.keys_tmp = off; off = align_up(off + 8 * (size_t)cap, 256);
    L.vals_tmp = off; off = align_up(off + 4 * (size_t)cap, 256);
    const size_t sort_tiles = (size_t)((cap + SORT_TILE - 1) / SORT_TILE);
    L.sort_status = off; off = align_up(off + 4 * (size_t)RADIX * sort_tiles * (size_t)num_passes_for(num_tiles), 256);
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

// ---------------------------------------------------------------------------------------------
// emit: scan + replicate + assign tile id + digit histograms
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(EMIT_THREADS)
emit_kernel(int64_t N, int TW, int num_passes, int64_t capacity, const float* __restrict__ depth,
            const int4* __restrict__ rect, const uint32_t* __restrict__ tcount, Header* __restrict__ hdr,
            unsigned long long* __restrict__ scan_status, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals) {
    __shared__ uint32_t s_off[EMIT_THREADS + 1];     // exclusive pair offsets of the block's Gaussians
    __shared__ int s_x0[EMIT_THREADS], s_y0[EMIT_THREADS], s_w[EMIT_THREADS];
    __shared__ uint32_t s_dbits[EMIT_THREADS];
    __shared__ uint32_t s_warp[EMIT_THREADS / 32];
    __shared__ uint32_t s_hist[MAX_PASSES * RADIX];
    __shared__ uint32_t s_block;
    __shared__ unsigned long long s_base;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_block = atomicAdd(&hdr->emit_ticket, 1u);   // ticket order = look-back order
    for (int b = tid; b < num_passes * RADIX; b += EMIT_THREADS) s_hist[b] = 0u;
    __syncthreads();
    const uint32_t block = s_block;
    const int64_t i = (int64_t)block * EMIT_THREADS + tid;

    uint32_t tc = 0;
    if (i < N) tc = tcount[i];
    if (tc) {
        const int4 r = rect[i];
        const uint32_t db = __float_as_uint(depth[i]);
        s_x0[tid] = r.x; s_y0[tid] = r.y; s_w[tid] = r.z - r.x; s_dbits[tid] = db;
#pragma unroll
        for (int d = 0; d < 4; ++d) atomicAdd(&s_hist[d * RADIX + ((db >> (8 * d)) & 255u)], tc);
    }
    // block exclusive scan of tc
    uint32_t incl = tc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint32_t wbase = 0, btotal = 0;
#pragma unroll
    for (int w = 0; w < EMIT_THREADS / 32; ++w) {
        const uint32_t v = s_warp[w];
        if (w < warp) wbase += v;
        btotal += v;
    }
    s_off[tid] = wbase + incl - tc;
    if (tid == 0) {
        s_off[EMIT_THREADS] = btotal;
        // decoupled look-back: publish the block aggregate, sum predecessors until an inclusive prefix
        unsigned long long excl = 0;
        if (block == 0) {
            st_relaxed64(&scan_status[0], SFLAG_INCLUSIVE | (unsigned long long)btotal);
        } else {
            st_relaxed64(&scan_status[block], SFLAG_PARTIAL | (unsigned long long)btotal);
            int64_t t = (int64_t)block - 1;
            while (true) {
                unsigned long long s;
                do { s = ld_relaxed64(&scan_status[t]); } while ((s & SFLAG_MASK) == 0);
                excl += s & ~SFLAG_MASK;
                if ((s & SFLAG_MASK) == SFLAG_INCLUSIVE) break;
                --t;
            }
            st_relaxed64(&scan_status[block], SFLAG_INCLUSIVE | (excl + btotal));
        }
        s_base = excl;
        if ((int64_t)(block + 1) * EMIT_THREADS >= N) hdr->total_pairs = excl + btotal;   // last block: I
    }
    __syncthreads();
    const unsigned long long base = s_base;
    // load-balanced emission: pair j of the block belongs to the last Gaussian g with s_off[g] <= j
    const uint32_t rounds = (btotal + EMIT_THREADS - 1) / EMIT_THREADS;
    for (uint32_t it = 0; it < rounds; ++it) {
        const uint32_t j = it * EMIT_THREADS + tid;
        const bool valid = j < btotal;
        uint32_t tile = 0;
        if (valid) {
            int lo = 0, hi = EMIT_THREADS;            // invariant: s_off[lo] <= j < s_off[hi]
#pragma unroll
            for (int s = 0; s < 8; ++s) {
                const int mid = (lo + hi) >> 1;
                if (s_off[mid] <= j) lo = mid; else hi = mid;
            }
            const uint32_t r = j - s_off[lo];
            const uint32_t w = (uint32_t)s_w[lo];
            const uint32_t ry = r / w, rx = r - ry * w;
            tile = (uint32_t)(s_y0[lo] + (int)ry) * (uint32_t)TW + (uint32_t)(s_x0[lo] + (int)rx);
            const unsigned long long gpos = base + j;
            if (gpos < (unsigned long long)capacity) {
                keys[gpos] = ((uint64_t)tile << 32) | (uint64_t)s_dbits[lo];
                vals[gpos] = (uint32_t)((int64_t)block * EMIT_THREADS + lo);
            }
            atomicAdd(&s_hist[4 * RADIX + (tile & 255u)], 1u);   // consecutive tiles -> distinct banks
        }
        // higher tile digits are nearly warp-uniform: aggregate with match.any before the atomic
        for (int d = 5; d < num_passes; ++d) {
            const uint32_t dig = valid ? ((tile >> (8 * (d - 4))) & 255u) : 0xffffffffu;
            const uint32_t peers = __match_any_sync(0xffffffffu, dig);
            if (valid && (peers & ((1u << lane) - 1u)) == 0u) atomicAdd(&s_hist[d * RADIX + dig], (uint32_t)__popc(peers));
        }
    }
    __syncthreads();
    for (int b = tid; b < num_passes * RADIX; b += EMIT_THREADS) {
        const uint32_t v = s_hist[b];
        if (v) atomicAdd(&hdr->hist[b], v);
    }
}

// ---------------------------------------------------------------------------------------------
// onesweep digit pass
// ---------------------------------------------------------------------------------------------
struct SortSmem {
    uint64_t keys[SORT_TILE];
    uint32_t vals[SORT_TILE];
    uint32_t warp_hist[SORT_WARPS][RADIX];
    uint32_t cta_excl[RADIX];     // exclusive digit offsets inside the tile
    uint32_t gbase[RADIX];        // global position of digit d's first key of this tile, minus cta_excl[d]
    uint32_t scan_tmp[SORT_WARPS];
    uint32_t tile_id;
};

__global__ void __launch_bounds__(SORT_THREADS)
onesweep_kernel(uint32_t I, int pass, const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, Header* __restrict__ hdr,
                uint32_t* __restrict__ status /* [tiles][RADIX] of this pass */) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem& S = *reinterpret_cast<SortSmem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int shift = pass * RADIX_BITS;

    if (tid == 0) S.tile_id = atomicAdd(&hdr->sort_ticket[pass], 1u);
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) S.warp_hist[w][tid] = 0u;    // SORT_THREADS == RADIX
    __syncthreads();
    const uint32_t tile = S.tile_id;
    const uint32_t tile_base = tile * (uint32_t)SORT_TILE;
    const uint32_t tile_n = min((uint32_t)SORT_TILE, I - tile_base);

    // warp-striped load: item `it` of lane l of warp w sits at tile_base + w*32*IPT + it*32 + l
    uint64_t key[SORT_IPT];
    uint32_t val[SORT_IPT];
    const uint32_t wofs = (uint32_t)warp * 32u * SORT_IPT + (uint32_t)lane;
#pragma unroll
    for (int it = 0; it < SORT_IPT; ++it) {
        const uint32_t loc = wofs + (uint32_t)it * 32u;
        if (loc < tile_n) {
            key[it] = keys_in[tile_base + loc];
            val[it] = vals_in[tile_base + loc];
        } else {
            key[it] = ~0ull;       // padding: highest digit, ranks after every real key of the tile
            val[it] = 0u;
        }
    }
    // stable in-warp ranking (match.any): rank = #earlier items of this warp with the same digit
    uint32_t rank[SORT_IPT];
    const uint32_t lt_mask = (1u << lane) - 1u;
#pragma unroll
    for (int it = 0; it < SORT_IPT; ++it) {
        const uint32_t d = (uint32_t)(key[it] >> shift) & (RADIX - 1);
        const uint32_t peers = __match_any_sync(0xffffffffu, d);
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
    if (tid == RADIX - 1) real_count -= (uint32_t)SORT_TILE - tile_n;
    // block exclusive scan over digits of `count` -> cta_excl; and of the global histogram -> bin base
    const uint32_t gh = hdr->hist[pass * RADIX + tid];
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
        while (true) {
            uint32_t s;
            do { s = ld_relaxed(p); } while ((s & FLAG_MASK) == 0u);
            excl_prev += s & VALUE_MASK;
            if ((s & FLAG_MASK) == FLAG_INCLUSIVE) break;
            p -= RADIX;
        }
        st_relaxed(my, FLAG_INCLUSIVE | (excl_prev + real_count));
    }
    S.gbase[tid] = bin_base + excl_prev - excl_c;
    __syncthreads();
    // scatter into shared memory in tile-sorted order
#pragma unroll
    for (int it = 0; it < SORT_IPT; ++it) {
        const uint32_t d = (uint32_t)(key[it] >> shift) & (RADIX - 1);
        const uint32_t pos = S.cta_excl[d] + S.warp_hist[warp][d] + rank[it];
        S.keys[pos] = key[it];
        S.vals[pos] = val[it];
    }
    __syncthreads();
    // coalesced runs to global memory (padding sits at positions >= tile_n)
#pragma unroll
    for (int it = 0; it < SORT_IPT; ++it) {
        const uint32_t p = (uint32_t)it * SORT_THREADS + (uint32_t)tid;
        if (p < tile_n) {
            const uint64_t k = S.keys[p];
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
    if (!bytes || N < 0 || pair_capacity < 0 || pair_capacity >= (1LL << 30) || num_tiles <= 0) return XPR_ERR_INVALID_ARG;
    *bytes = make_layout(N, pair_capacity, num_tiles).total;
    return XPR_OK;
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
    unsigned long long* scan_status = reinterpret_cast<unsigned long long*>(ws + L.scan_status);
    uint64_t* keys_tmp = reinterpret_cast<uint64_t*>(ws + L.keys_tmp);
    uint32_t* vals_tmp = reinterpret_cast<uint32_t*>(ws + L.vals_tmp);
    uint32_t* sort_status = reinterpret_cast<uint32_t*>(ws + L.sort_status);
    const int passes = num_passes_for(T);

    XPR_CUDA(cudaMemsetAsync(tile_ranges, 0, sizeof(uint32_t) * 2 * (size_t)T, st));
    *num_pairs_host = 0;
    if (N == 0) return XPR_OK;
    // header + scan status are contiguous: one memset
    XPR_CUDA(cudaMemsetAsync(ws + L.header, 0, L.keys_tmp - L.header, st));
    // an even number of passes ends in the buffer emission wrote to
    uint64_t* k0 = (passes % 2 == 0) ? keys_sorted : keys_tmp;
    uint32_t* v0 = (passes % 2 == 0) ? vals_sorted : vals_tmp;
    uint64_t* k1 = (passes % 2 == 0) ? keys_tmp : keys_sorted;
    uint32_t* v1 = (passes % 2 == 0) ? vals_tmp : vals_sorted;
    const unsigned emit_blocks = (unsigned)((N + EMIT_THREADS - 1) / EMIT_THREADS);
    emit_kernel<<<emit_blocks, EMIT_THREADS, 0, st>>>(N, TW, passes, pair_capacity, depth,
                                                      reinterpret_cast<const int4*>(tile_rect), tile_count, hdr,
                                                      scan_status, k0, v0);
    XPR_LAUNCH_CHECK();
    unsigned long long total = 0;
    XPR_CUDA(cudaMemcpyAsync(&total, &hdr->total_pairs, sizeof(total), cudaMemcpyDeviceToHost, st));
    XPR_CUDA(cudaStreamSynchronize(st));
    *num_pairs_host = (int64_t)total;
    if ((int64_t)total > pair_capacity) return XPR_ERR_CAPACITY;
    if (total == 0) return XPR_OK;
    const uint32_t I = (uint32_t)total;
    const unsigned sort_tiles = (I + SORT_TILE - 1) / SORT_TILE;
    XPR_CUDA(cudaMemsetAsync(sort_status, 0, sizeof(uint32_t) * (size_t)RADIX * sort_tiles * (size_t)passes, st));
    XPR_CUDA(cudaFuncSetAttribute(onesweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem)));
    for (int p = 0; p < passes; ++p) {
        onesweep_kernel<<<sort_tiles, SORT_THREADS, sizeof(SortSmem), st>>>(
            I, p, k0, v0, k1, v1, hdr, sort_status + (size_t)p * RADIX * sort_tiles);
        XPR_LAUNCH_CHECK();
        uint64_t* tk = k0; k0 = k1; k1 = tk;
        uint32_t* tv = v0; v0 = v1; v1 = tv;
    }
    ranges_kernel<<<(I + 255) / 256, 256, 0, st>>>(I, keys_sorted, tile_ranges);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}
