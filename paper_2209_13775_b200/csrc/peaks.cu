// peaks.cu -- micro-kernels that MEASURE the B200 peaks the roofline fractions of bench.py are quoted against
// (SURVEY.md 8.3 "Peaks to measure on the box before quoting any %": L2 read bandwidth sequential and random-sector over a
// 48 MB buffer, L1 hit bandwidth, random 32-byte HBM gather over a 2 GB buffer, FP32 / FP64 FMA throughput, launch latency).
// The paper's claim under re-examination is "primarily limited by memory bandwidth": these numbers say
// which level of the hierarchy binds each integrator.  One C-ABI call, lcs_measure_peak(kind, &value); synchronous; every
// kernel is timed with CUDA events after one warm-up launch, best of 3.
#include <math.h>

#include "lcs_internal.cuh"

namespace {

constexpr int kSMs = 148;

// ---- FP32 / FP64 FMA: 8 independent chains per thread
template <typename T> __global__ void __launch_bounds__(1024) fma_kernel(T *out, T a, T b, int iters)
{
    T x0 = (T)threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

__global__ void empty_kernel() {}

// ---- streaming copy (sanity against MEASURED_PEAKS.json) and sequential L2 read
__global__ void __launch_bounds__(512) copy_kernel(const float4 *__restrict__ src, float4 *__restrict__ dst, size_t n4)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) dst[i] = src[i];
}

__global__ void __launch_bounds__(512) seq_read_kernel(const float4 *__restrict__ p, float *out, size_t n4, int reps)
{
    float acc = 0.f;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int r = 0; r < reps; ++r)
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
            float4 v;
            asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p + i));   // L2 only
            acc += (v.x + v.y) + (v.z + v.w);
        }
    if (acc == 123.456f) out[0] = acc;
}

__device__ __forceinline__ uint32_t hash32(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

// ---- random 32-byte sector gather: every lane reads its own pseudo-random sector (one 256-bit load, L1 bypassed);
// 4 independent loads in flight per thread.  nsect must be a power of two.
__global__ void __launch_bounds__(256) sector_gather_kernel(const float *__restrict__ p, float *out, uint32_t nsect_mask, int iters)
{
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    float acc = 0.f;
    for (int it = 0; it < iters; it += 4) {
        float v[4][8];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const size_t s = hash32(t * 0x9e3779b9u + (uint32_t)(it + u)) & nsect_mask;
            asm volatile("ld.global.cg.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=f"(v[u][0]), "=f"(v[u][1]), "=f"(v[u][2]), "=f"(v[u][3]), "=f"(v[u][4]), "=f"(v[u][5]), "=f"(v[u][6]), "=f"(v[u][7])
                         : "l"(p + 8 * s));
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) acc += ((v[u][0] + v[u][1]) + (v[u][2] + v[u][3])) + ((v[u][4] + v[u][5]) + (v[u][6] + v[u][7]));
    }
    if (acc == 123.456f) out[0] = acc;
}

// ---- L1-resident LDG.256 gather.  MODE 0: the 4 lanes of a group read 4 consecutive records of one 128-byte line (the best
// case of the x-pair gather: 8 wavefronts per request); MODE 1: every lane of a group reads the SAME record; MODE 2: every
// lane reads a record in a line of its own (32 wavefronts per request).  The buffer (64 KB) stays in L1.
template <int MODE> __global__ void __launch_bounds__(256) l1_gather_kernel(const float *__restrict__ rec, float *out, int iters)
{
    constexpr uint32_t kRecMask = 2048 - 1;                 // 2048 records x 32 B = 64 KB
    const uint32_t lane = threadIdx.x & 31, warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    float acc = 0.f;
    for (int it = 0; it < iters; it += 4) {
        float v[4][8];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t r0 = hash32(warp * 0x9e3779b9u + (uint32_t)(it + u));
            uint32_t r;
            if (MODE == 0) r = ((hash32(r0 + (lane >> 2)) << 2) + (lane & 3)) & kRecMask;
            else if (MODE == 1) r = (hash32(r0 + (lane >> 2)) << 2) & kRecMask;
            else if (MODE == 2) r = ((hash32(r0 + lane) << 2)) & kRecMask;
            else if (MODE == 3) r = (r0 << 2) & kRecMask;                                    // the whole warp reads one record
            else if (MODE == 4) r = ((r0 << 2) + (lane & 3)) & kRecMask;                     // ... the 4 records of one line
            else r = ((hash32(r0 + (lane >> 4)) << 2) + (lane & 3)) & kRecMask;             // ... two lines, 16 lanes each
            asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=f"(v[u][0]), "=f"(v[u][1]), "=f"(v[u][2]), "=f"(v[u][3]), "=f"(v[u][4]), "=f"(v[u][5]), "=f"(v[u][6]), "=f"(v[u][7])
                         : "l"(rec + 8 * r));
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) acc += ((v[u][0] + v[u][1]) + (v[u][2] + v[u][3])) + ((v[u][4] + v[u][5]) + (v[u][6] + v[u][7]));
    }
    if (acc == 123.456f) out[0] = acc;
}

// ---- shared-memory LDS.128 reads.  MODE 0: lane L reads the 16-byte chunk base + L (contiguous, the conflict-free
// baseline).  MODE 1: lane L reads the 32-byte record base + L as two LDS.128 (lo halves, then hi halves: a 32-byte stride,
// so only half of the banks are used per instruction).  MODE 2: as 1 with the 16-byte chunks XOR-swizzled the way a TMA
// tensor map with CU_TENSOR_MAP_SWIZZLE_32B lays them out (chunk ^= (chunk >> 3) & 1).  MODE 3: as 2, the 4 lanes of a
// group reading the same record (broadcast).
__device__ __forceinline__ float4 lds128(const float4 *p)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"((uint32_t)__cvta_generic_to_shared(p)));
    return v;
}

template <int MODE> __global__ void __launch_bounds__(256) smem_gather_kernel(float *out, int iters)
{
    __shared__ float4 tile[2 * 1024];                       // 1024 records x 32 B = 32 KB
    for (int i = threadIdx.x; i < 2 * 1024; i += blockDim.x) tile[i] = make_float4((float)i, 1.f, 2.f, 3.f);
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float acc = 0.f;
    uint32_t base = warp * 37u;
    for (int it = 0; it < iters; it += 4) {
        float4 a[4], b[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            base = (base + 101u) & 1023u;
            if (MODE == 0) {
                const uint32_t c = (2u * base + lane) & 2047u;
                a[u] = lds128(tile + c);
                b[u] = lds128(tile + ((c + 32u) & 2047u));
            } else {
                const uint32_t r = (base + (MODE == 3 ? (lane & ~3u) : lane)) & 1023u;
                uint32_t c0 = 2u * r, c1 = 2u * r + 1u;
                if (MODE >= 2) { c0 ^= (c0 >> 3) & 1u; c1 ^= (c1 >> 3) & 1u; }
                a[u] = lds128(tile + c0);
                b[u] = lds128(tile + c1);
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)       // every component is consumed: ptxas narrows a vector load whose outputs are partly dead
            acc += ((a[u].x + a[u].y) + (a[u].z + a[u].w)) + ((b[u].x + b[u].y) + (b[u].z + b[u].w));
    }
    if (acc == 123.456f) out[0] = acc;
}

template <typename F> lcs_status time_best(F launch, double *ms_out)
{
    cudaEvent_t e0, e1;
    LCS_CUDA_OK(cudaEventCreate(&e0));
    LCS_CUDA_OK(cudaEventCreate(&e1));
    launch();                                               // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0, 0);
        launch();
        cudaEventRecord(e1, 0);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { lcs_set_error("peak kernel failed: %s", cudaGetErrorString(e)); cudaEventDestroy(e0); cudaEventDestroy(e1); return LCS_ERR_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        best = ms < best ? ms : best;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *ms_out = best;
    return LCS_OK;
}

}  // namespace

extern "C" lcs_status lcs_measure_peak(int32_t kind, double *value)
{
    if (!value) { lcs_set_error("null argument"); return LCS_ERR_INVALID_ARG; }
    *value = 0.0;
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0) { lcs_set_error("no CUDA device: liblcs has no CPU fallback"); return LCS_ERR_CUDA; }
    double ms = 0.0;
    lcs_status rc = LCS_OK;
    float *out = nullptr;
    LCS_CUDA_OK(cudaMalloc((void **)&out, (size_t)kSMs * 8 * 1024 * 8));
    void *buf = nullptr, *buf2 = nullptr;
    auto done = [&](lcs_status r) { cudaFree(out); if (buf) cudaFree(buf); if (buf2) cudaFree(buf2); return r; };
    switch (kind) {
    case LCS_PEAK_FP32_FMA: {
        const int iters = 20000;
        rc = time_best([&] { LCS_LAUNCH((fma_kernel<float>), kSMs * 8, 1024, 0, 0, out, 1.0001f, 0.5f, iters); }, &ms);
        *value = 2.0 * 8 * iters * (double)kSMs * 8 * 1024 / (ms * 1e-3) / 1e12;
        break;
    }
    case LCS_PEAK_FP64_FMA: {
        const int iters = 2000;
        rc = time_best([&] { LCS_LAUNCH((fma_kernel<double>), kSMs * 8, 1024, 0, 0, (double *)out, 1.0001, 0.5, iters); }, &ms);
        *value = 2.0 * 8 * iters * (double)kSMs * 8 * 1024 / (ms * 1e-3) / 1e12;
        break;
    }
    case LCS_PEAK_LAUNCH_US: {
        const int reps = 2000;
        rc = time_best([&] { for (int i = 0; i < reps; ++i) LCS_LAUNCH(empty_kernel, 1, 32, 0, 0); }, &ms);
        *value = ms * 1e3 / reps;
        break;
    }
    case LCS_PEAK_HBM_COPY: {
        const size_t bytes = (size_t)1 << 30;
        if (cudaMalloc(&buf, bytes) != cudaSuccess || cudaMalloc(&buf2, bytes) != cudaSuccess) { lcs_set_error("out of memory"); return done(LCS_ERR_OOM); }
        cudaMemset(buf, 0, bytes);
        rc = time_best([&] { LCS_LAUNCH(copy_kernel, kSMs * 8, 512, 0, 0, (const float4 *)buf, (float4 *)buf2, bytes / 16); }, &ms);
        *value = 2.0 * bytes / (ms * 1e-3) / 1e9;
        break;
    }
    case LCS_PEAK_L2_SEQ: {
        const size_t bytes = (size_t)48 << 20;
        const int reps = 50;
        if (cudaMalloc(&buf, bytes) != cudaSuccess) { lcs_set_error("out of memory"); return done(LCS_ERR_OOM); }
        cudaMemset(buf, 0, bytes);
        rc = time_best([&] { LCS_LAUNCH(seq_read_kernel, kSMs * 8, 512, 0, 0, (const float4 *)buf, out, bytes / 16, reps); }, &ms);
        *value = (double)reps * bytes / (ms * 1e-3) / 1e9;
        break;
    }
    case LCS_PEAK_L2_SECTOR:
    case LCS_PEAK_HBM_SECTOR: {
        const size_t bytes = kind == LCS_PEAK_L2_SECTOR ? (size_t)32 << 20 : (size_t)2 << 30;     // powers of two; 32 MB stays in the 126 MB L2
        const int iters = kind == LCS_PEAK_L2_SECTOR ? 512 : 128;
        const int blocks = kSMs * 32;
        if (cudaMalloc(&buf, bytes) != cudaSuccess) { lcs_set_error("out of memory"); return done(LCS_ERR_OOM); }
        cudaMemset(buf, 0, bytes);
        rc = time_best([&] { LCS_LAUNCH(sector_gather_kernel, blocks, 256, 0, 0, (const float *)buf, out, (uint32_t)(bytes / 32 - 1), iters); }, &ms);
        *value = 32.0 * blocks * 256 * iters / (ms * 1e-3) / 1e9;
        break;
    }
    case LCS_PEAK_L1_GATHER_LINE:
    case LCS_PEAK_L1_GATHER_SAME:
    case LCS_PEAK_L1_GATHER_SPREAD:
    case LCS_PEAK_L1_GATHER_WARP_SAME:
    case LCS_PEAK_L1_GATHER_WARP_LINE:
    case LCS_PEAK_L1_GATHER_WARP_2LINES: {
        const int iters = 2000, blocks = kSMs * 8;
        if (cudaMalloc(&buf, 64 << 10) != cudaSuccess) { lcs_set_error("out of memory"); return done(LCS_ERR_OOM); }
        cudaMemset(buf, 0, 64 << 10);
        if (kind == LCS_PEAK_L1_GATHER_LINE) rc = time_best([&] { LCS_LAUNCH((l1_gather_kernel<0>), blocks, 256, 0, 0, (const float *)buf, out, iters); }, &ms);
        else if (kind == LCS_PEAK_L1_GATHER_SAME) rc = time_best([&] { LCS_LAUNCH((l1_gather_kernel<1>), blocks, 256, 0, 0, (const float *)buf, out, iters); }, &ms);
        else if (kind == LCS_PEAK_L1_GATHER_SPREAD) rc = time_best([&] { LCS_LAUNCH((l1_gather_kernel<2>), blocks, 256, 0, 0, (const float *)buf, out, iters); }, &ms);
        else if (kind == LCS_PEAK_L1_GATHER_WARP_SAME) rc = time_best([&] { LCS_LAUNCH((l1_gather_kernel<3>), blocks, 256, 0, 0, (const float *)buf, out, iters); }, &ms);
        else if (kind == LCS_PEAK_L1_GATHER_WARP_LINE) rc = time_best([&] { LCS_LAUNCH((l1_gather_kernel<4>), blocks, 256, 0, 0, (const float *)buf, out, iters); }, &ms);
        else rc = time_best([&] { LCS_LAUNCH((l1_gather_kernel<5>), blocks, 256, 0, 0, (const float *)buf, out, iters); }, &ms);
        *value = 32.0 * blocks * 256 * iters / (ms * 1e-3) / 1e9;
        break;
    }
    case LCS_PEAK_SMEM_CONTIGUOUS:
    case LCS_PEAK_SMEM_RECORDS:
    case LCS_PEAK_SMEM_RECORDS_SWIZZLED:
    case LCS_PEAK_SMEM_RECORDS_SAME: {
        const int iters = 4000, blocks = kSMs * 6;
        if (kind == LCS_PEAK_SMEM_CONTIGUOUS) rc = time_best([&] { LCS_LAUNCH((smem_gather_kernel<0>), blocks, 256, 0, 0, out, iters); }, &ms);
        else if (kind == LCS_PEAK_SMEM_RECORDS) rc = time_best([&] { LCS_LAUNCH((smem_gather_kernel<1>), blocks, 256, 0, 0, out, iters); }, &ms);
        else if (kind == LCS_PEAK_SMEM_RECORDS_SWIZZLED) rc = time_best([&] { LCS_LAUNCH((smem_gather_kernel<2>), blocks, 256, 0, 0, out, iters); }, &ms);
        else rc = time_best([&] { LCS_LAUNCH((smem_gather_kernel<3>), blocks, 256, 0, 0, out, iters); }, &ms);
        *value = 32.0 * blocks * 256 * iters / (ms * 1e-3) / 1e9;
        break;
    }
    default:
        lcs_set_error("unknown peak kind %d", kind);
        return done(LCS_ERR_INVALID_ARG);
    }
    if (rc == LCS_OK && cudaGetLastError() != cudaSuccess) { lcs_set_error("peak kernel launch failed"); rc = LCS_ERR_CUDA; }
    return done(rc);
}
