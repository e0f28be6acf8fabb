// Device-wide exclusive prefix sum (reduce-then-scan, three kernels, recursive on the tile sums).
// out has n+1 entries: out[i] = Σ_{j<i} in[j], out[n] = total.  int64 accumulation.
// Hot-path step 4 of DESIGN.md ("scan + budget"); also used by the packer, the merge stage and assembly.
#pragma once

#include "common.cuh"

namespace fstc {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;                         // per thread
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;  // 2048 elements per block

__device__ __forceinline__ int64_t warp_incl_scan(int64_t v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int64_t t = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += t;
    }
    return v;
}

// Loads are warp-striped (coalesced): warp w of the block owns elements [w*256, w*256+256) of the tile,
// visited in 8 rounds of 32 consecutive elements.
template <typename InT>
__global__ void __launch_bounds__(SCAN_THREADS) scan_tile_sums(const InT *__restrict__ in, int64_t n,
                                                                int64_t *__restrict__ sums) {
    __shared__ int64_t wsum[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t base = static_cast<int64_t>(blockIdx.x) * SCAN_TILE + warp * (32 * SCAN_ITEMS);
    int64_t s = 0;
#pragma unroll
    for (int r = 0; r < SCAN_ITEMS; ++r) {
        int64_t i = base + r * 32 + lane;
        if (i < n) s += static_cast<int64_t>(in[i]);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if (lane == 0) wsum[warp] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        int64_t t = 0;
#pragma unroll
        for (int w = 0; w < SCAN_THREADS / 32; ++w) t += wsum[w];
        sums[blockIdx.x] = t;
    }
}

// tile_off: exclusive prefix of the tile sums (nullptr = single tile starting at 0).
template <typename InT>
__global__ void __launch_bounds__(SCAN_THREADS) scan_tile_down(const InT *in, int64_t n,
                                                                const int64_t *__restrict__ tile_off,
                                                                int64_t *out, bool write_total) {
    __shared__ int64_t wsum[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t base = static_cast<int64_t>(blockIdx.x) * SCAN_TILE + warp * (32 * SCAN_ITEMS);
    int64_t x[SCAN_ITEMS], ex[SCAN_ITEMS];
#pragma unroll
    for (int r = 0; r < SCAN_ITEMS; ++r) {
        int64_t i = base + r * 32 + lane;
        x[r] = (i < n) ? static_cast<int64_t>(in[i]) : 0;
    }
    int64_t carry = 0;
#pragma unroll
    for (int r = 0; r < SCAN_ITEMS; ++r) {
        int64_t inc = warp_incl_scan(x[r], lane);
        ex[r] = carry + inc - x[r];
        carry += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) wsum[warp] = carry;
    __syncthreads();
    int64_t off = tile_off ? tile_off[blockIdx.x] : 0;
    for (int w = 0; w < warp; ++w) off += wsum[w];
#pragma unroll
    for (int r = 0; r < SCAN_ITEMS; ++r) {
        int64_t i = base + r * 32 + lane;
        if (i < n) out[i] = off + ex[r];
    }
    if (write_total && blockIdx.x == gridDim.x - 1 && threadIdx.x == SCAN_THREADS - 1) {
        // last thread of the last tile: its running total covers the whole tile
        out[n] = off + carry;
    }
}

// out must have room for n+1 values.  in and out may alias only if InT is int64_t and in == out.
template <typename InT>
void exclusive_scan(Ctx &c, const InT *in, int64_t n, int64_t *out) {
    if (n <= 0) {
        FSTC_CUDA(cudaMemsetAsync(out, 0, sizeof(int64_t), c.stream));
        return;
    }
    const int64_t tiles = ceil_div(n, SCAN_TILE);
    if (tiles == 1) {
        scan_tile_down<InT><<<1, SCAN_THREADS, 0, c.stream>>>(in, n, nullptr, out, true);
        FSTC_LAUNCH_CHECK();
        c.n_launch += 1;
        return;
    }
    DBuf<int64_t> sums(c, tiles + 1);
    scan_tile_sums<InT><<<static_cast<unsigned>(tiles), SCAN_THREADS, 0, c.stream>>>(in, n, sums.p);
    FSTC_LAUNCH_CHECK();
    exclusive_scan<int64_t>(c, sums.p, tiles, sums.p);   // in place; sums[tiles] = total
    scan_tile_down<InT><<<static_cast<unsigned>(tiles), SCAN_THREADS, 0, c.stream>>>(in, n, sums.p, out, true);
    FSTC_LAUNCH_CHECK();
    c.n_launch += 2;
}

// Fused scan of two arrays of equal length (a: int64, b: uint32) in one pass over each: used once per BFS level for
// (raw arc counts, match counts).  outA / outB have n+1 entries each.
static __global__ void __launch_bounds__(SCAN_THREADS) scan2_tile_sums(const int64_t *__restrict__ a, const uint32_t *__restrict__ b,
                                                                 int64_t n, int64_t *__restrict__ sumsA,
                                                                 int64_t *__restrict__ sumsB) {
    __shared__ int64_t wa[SCAN_THREADS / 32], wb[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t base = static_cast<int64_t>(blockIdx.x) * SCAN_TILE + warp * (32 * SCAN_ITEMS);
    int64_t sa = 0, sb = 0;
#pragma unroll
    for (int r = 0; r < SCAN_ITEMS; ++r) {
        int64_t i = base + r * 32 + lane;
        if (i < n) { sa += a[i]; sb += b[i]; }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        sa += __shfl_xor_sync(0xffffffffu, sa, d);
        sb += __shfl_xor_sync(0xffffffffu, sb, d);
    }
    if (lane == 0) { wa[warp] = sa; wb[warp] = sb; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int64_t ta = 0, tb = 0;
#pragma unroll
        for (int w = 0; w < SCAN_THREADS / 32; ++w) { ta += wa[w]; tb += wb[w]; }
        sumsA[blockIdx.x] = ta; sumsB[blockIdx.x] = tb;
    }
}

static __global__ void __launch_bounds__(SCAN_THREADS) scan2_tile_down(const int64_t *__restrict__ a, const uint32_t *__restrict__ b,
                                                                 int64_t n, const int64_t *__restrict__ offA,
                                                                 const int64_t *__restrict__ offB, int64_t *__restrict__ outA,
                                                                 int64_t *__restrict__ outB) {
    __shared__ int64_t wa[SCAN_THREADS / 32], wb[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t base = static_cast<int64_t>(blockIdx.x) * SCAN_TILE + warp * (32 * SCAN_ITEMS);
    int64_t ea[SCAN_ITEMS], eb[SCAN_ITEMS];
    int64_t ca = 0, cb = 0;
#pragma unroll
    for (int r = 0; r < SCAN_ITEMS; ++r) {
        int64_t i = base + r * 32 + lane;
        int64_t xa = (i < n) ? a[i] : 0, xb = (i < n) ? static_cast<int64_t>(b[i]) : 0;
        int64_t ia = warp_incl_scan(xa, lane), ib = warp_incl_scan(xb, lane);
        ea[r] = ca + ia - xa; eb[r] = cb + ib - xb;
        ca += __shfl_sync(0xffffffffu, ia, 31);
        cb += __shfl_sync(0xffffffffu, ib, 31);
    }
    if (lane == 0) { wa[warp] = ca; wb[warp] = cb; }
    __syncthreads();
    int64_t oa = offA ? offA[blockIdx.x] : 0, ob = offB ? offB[blockIdx.x] : 0;
    for (int w = 0; w < warp; ++w) { oa += wa[w]; ob += wb[w]; }
#pragma unroll
    for (int r = 0; r < SCAN_ITEMS; ++r) {
        int64_t i = base + r * 32 + lane;
        if (i < n) { outA[i] = oa + ea[r]; outB[i] = ob + eb[r]; }
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == SCAN_THREADS - 1) { outA[n] = oa + ca; outB[n] = ob + cb; }
}

inline void exclusive_scan2(Ctx &c, const int64_t *a, const uint32_t *b, int64_t n, int64_t *outA, int64_t *outB) {
    if (n <= 0) {
        FSTC_CUDA(cudaMemsetAsync(outA, 0, sizeof(int64_t), c.stream));
        FSTC_CUDA(cudaMemsetAsync(outB, 0, sizeof(int64_t), c.stream));
        return;
    }
    const int64_t tiles = ceil_div(n, SCAN_TILE);
    if (tiles == 1) {
        scan2_tile_down<<<1, SCAN_THREADS, 0, c.stream>>>(a, b, n, nullptr, nullptr, outA, outB);
        FSTC_LAUNCH_CHECK();
        c.n_launch += 1;
        return;
    }
    DBuf<int64_t> sa(c, tiles + 1), sb(c, tiles + 1);
    scan2_tile_sums<<<static_cast<unsigned>(tiles), SCAN_THREADS, 0, c.stream>>>(a, b, n, sa.p, sb.p);
    FSTC_LAUNCH_CHECK();
    exclusive_scan<int64_t>(c, sa.p, tiles, sa.p);
    exclusive_scan<int64_t>(c, sb.p, tiles, sb.p);
    scan2_tile_down<<<static_cast<unsigned>(tiles), SCAN_THREADS, 0, c.stream>>>(a, b, n, sa.p, sb.p, outA, outB);
    FSTC_LAUNCH_CHECK();
    c.n_launch += 2;
}

}  // namespace fstc
