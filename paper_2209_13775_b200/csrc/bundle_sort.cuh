// bundle_sort.cuh -- re-bundling of tracers by cell: a device counting sort (histogram, exclusive scan,
// scatter) over fixed-size tracer records.  Private to liblcs.so.
//
// Why: the paper notes that tracers "disperse" so that sorting the velocity data gave no gain
// and cites re-bundling of tracers for coherence (ref [6]).  On B200 the integrator is bound by
// L1 wavefronts (one 128-byte line per cycle per SM): a 256-bit gather costs one wavefront per distinct line that each
// group of 4 lanes touches -- 8 per warp when neighbouring lanes sit in the same or x-neighbouring cells, up to 32 when
// the tracers of a warp are dispersed.  Tracer
// results do not depend on the order (every tracer is independent), so the scatter may place
// equal keys in any order (atomic slot allocation).
#pragma once
#include "lcs_internal.cuh"

namespace bundle {

constexpr int kScanBlock = 1024;
constexpr int kScanItems = 4;                    // per thread
constexpr int kScanTile = kScanBlock * kScanItems;
constexpr uint32_t kDropKey = 0xffffffffu;         // a record with this key is not counted and not scattered: it leaves the set

// spread the low 10 bits of v so that there are two zero bits between consecutive bits
__host__ __device__ __forceinline__ uint32_t spread3(uint32_t v)
{
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000ffu;
    v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}
__host__ __device__ __forceinline__ uint32_t spread2(uint32_t v)
{
    v &= 0xffffu;
    v = (v | (v << 8)) & 0x00ff00ffu;
    v = (v | (v << 4)) & 0x0f0f0f0fu;
    v = (v | (v << 2)) & 0x33333333u;
    v = (v | (v << 1)) & 0x55555555u;
    return v;
}
template <int DIM> __host__ __device__ __forceinline__ uint32_t morton(const int *c)
{
    if constexpr (DIM == 2) return spread2((uint32_t)c[0]) | (spread2((uint32_t)c[1]) << 1);
    else return spread3((uint32_t)c[0]) | (spread3((uint32_t)c[1]) << 1) | (spread3((uint32_t)c[2]) << 2);
}

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, v, d);
        if ((threadIdx.x & 31) >= d) v += t;
    }
    return v;
}

// block-wide exclusive scan of one value per thread (kScanBlock threads); returns the exclusive prefix and
// the block total through *total
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t *total)
{
    __shared__ uint32_t wsum[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t inc = warp_incl_scan(v);
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        uint32_t s = wsum[lane];
        uint32_t si = warp_incl_scan(s);
        wsum[lane] = si - s;
        if (lane == 31) wsum[31] = si - s, *total = si;
    }
    __syncthreads();
    uint32_t r = wsum[wid] + inc - v;
    __syncthreads();
    return r;
}

// pass 1: sum of every tile of kScanTile counters
static __global__ void __launch_bounds__(kScanBlock) scan_tile_sums_kernel(const uint32_t *__restrict__ cnt, int64_t nbins,
                                                                           uint32_t *__restrict__ tile_sum)
{
    __shared__ uint32_t tot;
    int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k)
        if (base + k < nbins) s += cnt[base + k];
    block_excl_scan(s, &tot);
    if (threadIdx.x == 0) tile_sum[blockIdx.x] = tot;
}

// pass 2: one block turns the tile sums into exclusive tile offsets
static __global__ void __launch_bounds__(kScanBlock) scan_tile_offsets_kernel(uint32_t *__restrict__ tile_sum, int64_t ntiles)
{
    __shared__ uint32_t tot;
    __shared__ uint32_t carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int64_t base = 0; base < ntiles; base += kScanBlock) {
        int64_t i = base + threadIdx.x;
        uint32_t v = i < ntiles ? tile_sum[i] : 0u;
        uint32_t ex = block_excl_scan(v, &tot);
        uint32_t carry = carry_s;
        if (i < ntiles) tile_sum[i] = carry + ex;
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + tot;
        __syncthreads();
    }
}

// pass 3: counters -> exclusive offsets, in place
static __global__ void __launch_bounds__(kScanBlock) scan_apply_kernel(uint32_t *__restrict__ cnt, int64_t nbins,
                                                                       const uint32_t *__restrict__ tile_off)
{
    __shared__ uint32_t tot;
    int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    uint32_t v[kScanItems], s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) { v[k] = base + k < nbins ? cnt[base + k] : 0u; s += v[k]; }
    uint32_t ex = block_excl_scan(s, &tot) + tile_off[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < nbins) cnt[base + k] = ex;
        ex += v[k];
    }
}

// histogram increment; the last bin (finished tracers, possibly most of the set) is aggregated per warp so that its
// single counter is hit once per warp instead of once per tracer
__device__ __forceinline__ void count_key(uint32_t *__restrict__ cnt, uint32_t k, uint32_t last_bin)
{
    const unsigned active = __activemask();
    const unsigned parked = __ballot_sync(active, k == last_bin);
    if (k != last_bin) atomicAdd(cnt + k, 1u);
    else if ((threadIdx.x & 31) == __ffs(parked) - 1) atomicAdd(cnt + last_bin, (uint32_t)__popc(parked));
}

// scatter: record i goes to the next free slot of its key (warp-aggregated for the last bin)
template <typename REC>
static __global__ void __launch_bounds__(256) scatter_kernel(const REC *__restrict__ src, const uint32_t *__restrict__ key,
                                                             uint32_t *__restrict__ offset, int64_t n, uint32_t last_bin,
                                                             REC *__restrict__ dst)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    static_assert(sizeof(REC) % 16 == 0, "tracer records are multiples of 16 bytes");
    constexpr int NQ = sizeof(REC) / 16;
    int4 q[NQ];
    const int4 *s = reinterpret_cast<const int4 *>(src + i);
#pragma unroll
    for (int k = 0; k < NQ; ++k) q[k] = s[k];
    const uint32_t k = key[i];
    if (k == kDropKey) return;
    const unsigned active = __activemask();
    const unsigned parked = __ballot_sync(active, k == last_bin);
    uint32_t pos;
    if (k != last_bin) {
        pos = atomicAdd(offset + k, 1u);
    } else {
        const int lane = threadIdx.x & 31, leader = __ffs(parked) - 1;
        uint32_t base = 0;
        if (lane == leader) base = atomicAdd(offset + last_bin, (uint32_t)__popc(parked));
        base = __shfl_sync(parked, base, leader);
        pos = base + (uint32_t)__popc(parked & ((1u << lane) - 1u));
    }
    int4 *d = reinterpret_cast<int4 *>(dst + pos);
#pragma unroll
    for (int k2 = 0; k2 < NQ; ++k2) d[k2] = q[k2];
}

static inline size_t scratch_bytes(int64_t n, int64_t nbins)
{
    auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
    int64_t ntiles = (nbins + kScanTile - 1) / kScanTile;
    return up((size_t)n * 4) + up((size_t)nbins * 4) + up((size_t)ntiles * 4);
}

// key[] (n) and cnt[] (nbins, already holding the histogram) -> dst = src sorted by key.  All on `st`.
template <typename REC>
static inline void sort_records(const REC *src, REC *dst, const uint32_t *key, uint32_t *cnt, uint32_t *tile, int64_t n, int64_t nbins,
                                cudaStream_t st)
{
    int64_t ntiles = (nbins + kScanTile - 1) / kScanTile;
    LCS_LAUNCH(scan_tile_sums_kernel, (unsigned)ntiles, kScanBlock, 0, st, cnt, nbins, tile);
    LCS_LAUNCH(scan_tile_offsets_kernel, 1, kScanBlock, 0, st, tile, ntiles);
    LCS_LAUNCH(scan_apply_kernel, (unsigned)ntiles, kScanBlock, 0, st, cnt, nbins, tile);
    LCS_LAUNCH((scatter_kernel<REC>), lcs_blocks(n, 256), 256, 0, st, src, key, cnt, n, (uint32_t)(nbins - 1), dst);
}

}  // namespace bundle
