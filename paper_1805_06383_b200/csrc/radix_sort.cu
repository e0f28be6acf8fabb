// Hand-written stable LSD radix sort of 16-byte records (step 7; also the packer
// and nothing else).  The paper sorts 64-bit packed keys with a library sort; here the
// sort is our own: per pass an upsweep (per-block digit histogram), an exclusive scan of the
// digit-major histogram, and a downsweep that ranks each tile stably with warp match-any and scatters
// whole 16-byte records.  Blocks own contiguous runs of tiles, so the histogram is 256 x grid counters.
#include "internal.h"
#include "scan.cuh"

namespace fstc {

namespace {

constexpr int RS_THREADS = 256;
constexpr int RS_WARPS = RS_THREADS / 32;
constexpr int RS_ITEMS = 8;
constexpr int RS_TILE = RS_THREADS * RS_ITEMS;   // 2048 records = 32 KB per tile
constexpr int RS_RADIX = 256;

// A record sorts as the number (z << key_bits) | key; a digit is `mask` at bit `shift` of it and may straddle the two.
// `word` carries key_bits.
__device__ __forceinline__ uint32_t digit_of(const uint4 &r, int key_bits, int shift, uint32_t mask) {
    const uint64_t k = (static_cast<uint64_t>(r.y) << 32) | r.x;
    const uint64_t lo = shift < key_bits ? k >> shift : 0ull;
    const uint64_t hi = shift <= key_bits ? (key_bits - shift < 64 ? static_cast<uint64_t>(r.z) << (key_bits - shift) : 0ull)
                                          : static_cast<uint64_t>(r.z) >> (shift - key_bits);
    return static_cast<uint32_t>(lo | hi) & mask;
}

__global__ void __launch_bounds__(RS_THREADS) rs_upsweep(const uint4 *__restrict__ in, int64_t n,
                                                          int64_t tiles_per_block, int word, int shift,
                                                          uint32_t mask, uint32_t *__restrict__ hist) {
    __shared__ uint32_t h[RS_WARPS][RS_RADIX];   // warp-private bins: no inter-warp contention
    for (int i = threadIdx.x; i < RS_WARPS * RS_RADIX; i += RS_THREADS) (&h[0][0])[i] = 0;
    __syncthreads();
    const int warp = threadIdx.x >> 5;
    const int64_t lo = static_cast<int64_t>(blockIdx.x) * tiles_per_block * RS_TILE;
    int64_t hi = lo + tiles_per_block * RS_TILE;
    if (hi > n) hi = n;
    for (int64_t i = lo + threadIdx.x; i < hi; i += RS_THREADS) {
        uint4 r = __ldg(in + i);
        atomicAdd(&h[warp][digit_of(r, word, shift, mask)], 1u);
    }
    __syncthreads();
    for (int d = threadIdx.x; d < RS_RADIX; d += RS_THREADS) {
        uint32_t s = 0;
#pragma unroll
        for (int w = 0; w < RS_WARPS; ++w) s += h[w][d];
        hist[static_cast<int64_t>(d) * gridDim.x + blockIdx.x] = s;
    }
}

__global__ void __launch_bounds__(RS_THREADS) rs_downsweep(const uint4 *__restrict__ in, uint4 *__restrict__ out,
                                                            int64_t n, int64_t tiles_per_block, int word, int shift,
                                                            uint32_t mask, const int64_t *__restrict__ offs) {
    __shared__ int64_t base[RS_RADIX];            // next free output slot of every digit for this block
    __shared__ uint32_t wcnt[RS_WARPS][RS_RADIX]; // per-warp digit counts of the current tile -> warp offsets
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t lt = (1u << lane) - 1u;
    for (int d = threadIdx.x; d < RS_RADIX; d += RS_THREADS)
        base[d] = offs[static_cast<int64_t>(d) * gridDim.x + blockIdx.x];
    const int64_t first = static_cast<int64_t>(blockIdx.x) * tiles_per_block;
    for (int64_t t = 0; t < tiles_per_block; ++t) {
        const int64_t tile_base = (first + t) * RS_TILE;
        if (tile_base >= n) break;
        for (int i = threadIdx.x; i < RS_WARPS * RS_RADIX; i += RS_THREADS) (&wcnt[0][0])[i] = 0;
        __syncthreads();
        uint4 rec[RS_ITEMS];
        uint32_t dig[RS_ITEMS], rnk[RS_ITEMS];
        const int64_t wbase = tile_base + warp * (32 * RS_ITEMS);
#pragma unroll
        for (int r = 0; r < RS_ITEMS; ++r) {
            int64_t i = wbase + r * 32 + lane;
            if (i < n) rec[r] = __ldg(in + i);
        }
#pragma unroll
        for (int r = 0; r < RS_ITEMS; ++r) {     // records of a warp are ranked in input order: stable
            int64_t i = wbase + r * 32 + lane;
            const bool valid = i < n;
            dig[r] = valid ? digit_of(rec[r], word, shift, mask) : 0xFFFFu;
            uint32_t peers = __match_any_sync(0xffffffffu, dig[r]);
            uint32_t my = __popc(peers & lt);
            uint32_t prev = valid ? wcnt[warp][dig[r]] : 0;
            __syncwarp();
            if (valid && my == 0) wcnt[warp][dig[r]] = prev + __popc(peers);
            __syncwarp();
            rnk[r] = prev + my;
        }
        __syncthreads();
        uint32_t tile_total = 0;
        {   // exclusive scan over the warps, one digit per thread (RS_THREADS == RS_RADIX)
            const int d = threadIdx.x;
#pragma unroll
            for (int w = 0; w < RS_WARPS; ++w) {
                uint32_t c = wcnt[w][d];
                wcnt[w][d] = tile_total;
                tile_total += c;
            }
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < RS_ITEMS; ++r) {
            if (dig[r] != 0xFFFFu) {
                int64_t pos = base[dig[r]] + wcnt[warp][dig[r]] + rnk[r];
                out[pos] = rec[r];
            }
        }
        __syncthreads();
        base[threadIdx.x] += tile_total;
    }
}

}  // namespace

std::vector<SortPass> make_sort_passes(int key_bits, int z_bits, int from_bit) {
    std::vector<SortPass> p;
    const int total = key_bits + z_bits;
    for (int s = from_bit; s < total; s += 8) p.push_back(SortPass{key_bits, s, total - s < 8 ? total - s : 8});
    return p;
}

uint4 *radix_sort_records(Ctx &c, uint4 *a, uint4 *b, int64_t n, const std::vector<SortPass> &passes) {
    static_assert(RS_THREADS == RS_RADIX, "one digit per thread in the warp-offset scan");
    if (n <= 1 || passes.empty()) return a;
    const int64_t tiles = ceil_div(n, RS_TILE);
    int64_t grid = tiles < static_cast<int64_t>(c.n_sm) * 4 ? tiles : static_cast<int64_t>(c.n_sm) * 4;
    const int64_t tpb = ceil_div(tiles, grid);
    grid = ceil_div(tiles, tpb);
    DBuf<uint32_t> hist(c, RS_RADIX * grid);
    DBuf<int64_t> offs(c, RS_RADIX * grid + 1);
    uint4 *src = a, *dst = b;
    for (const SortPass &p : passes) {
        const uint32_t mask = (1u << p.bits) - 1u;
        rs_upsweep<<<static_cast<unsigned>(grid), RS_THREADS, 0, c.stream>>>(src, n, tpb, p.word, p.shift, mask, hist.p);
        FSTC_LAUNCH_CHECK();
        exclusive_scan<uint32_t>(c, hist.p, RS_RADIX * grid, offs.p);
        rs_downsweep<<<static_cast<unsigned>(grid), RS_THREADS, 0, c.stream>>>(src, dst, n, tpb, p.word, p.shift, mask,
                                                                              offs.p);
        FSTC_LAUNCH_CHECK();
        c.n_launch += 2;
        uint4 *t = src; src = dst; dst = t;
    }
    return src;
}

}  // namespace fstc
