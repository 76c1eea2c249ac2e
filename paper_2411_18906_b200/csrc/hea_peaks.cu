// hea_peaks.cu -- micro-benchmarks for the roofline denominators that MEASURED_PEAKS.json does not hold (SURVEY 8d:
// "L2 random-sector GB/s, shared-memory gather rate, fp64/int issue rates must be measured on the box").  Product code
// (sm_100a); nothing from oracle/.  Each kernel runs one resource flat out with the access pattern the MC / recount
// kernels have; hea_measure_peaks times them with CUDA events and reports rates for the whole chip.
//
//   [0] random shared-memory byte gathers / s      LDS.U8 at pseudo-random addresses of a 128 KB array, 32 lanes -> random
//                                                  banks (the neighbour-species gathers of mc_halo_kernel)
//   [1] shared-memory wavefronts / s               conflict-free LDS.32: the data-pipe limit the gathers are measured against
//   [2] INT32 ALU-pipe thread-instructions / s     independent LOP3 chains
//   [3] FMA-pipe integer thread-instructions / s   independent IMAD chains
//   [4] mixed issue thread-instructions / s        LOP3 and IMAD interleaved (both pipes busy): the issue ceiling
//   [5] fp64 thread-instructions / s               independent DADD / DMUL chains (the D6 objective)
//   [6] L2 random 32-byte sectors, GB/s            LDG of random sectors of a 64 MB array (occupancy read through L2)
//   [7] SM clock in MHz assumed for derived figures (device attribute)
#include <cstdint>
#include <cuda_runtime.h>

namespace hea {

namespace {

constexpr int kPeakThreads = 512;

__global__ void __launch_bounds__(kPeakThreads) peak_lds_u8_kernel(uint32_t* out, int iters)
{
    extern __shared__ uint8_t s_buf[];
    constexpr uint32_t kBytes = 128u * 1024u;
    for (uint32_t i = threadIdx.x; i < kBytes; i += blockDim.x) s_buf[i] = (uint8_t)(i * 2654435761u >> 24);
    __syncthreads();
    uint32_t x = threadIdx.x * 2654435761u + blockIdx.x * 40503u + 12345u, acc = 0;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            x = x * 1664525u + 1013904223u;                   // one IMAD per gather: the address stream
            acc += s_buf[x >> 15];                            // 17 random bits -> 128 KB
        }
    }
    if (acc == 0xFFFFFFFFu) out[0] = acc;
}

__global__ void __launch_bounds__(kPeakThreads) peak_lds_wave_kernel(uint32_t* out, int iters)
{
    extern __shared__ uint8_t s_buf[];
    uint32_t* s32 = reinterpret_cast<uint32_t*>(s_buf);
    for (uint32_t i = threadIdx.x; i < 32u * 1024u; i += blockDim.x) s32[i] = i;
    __syncthreads();
    uint32_t idx = threadIdx.x, acc = 0;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            acc += s32[(idx + 32u * u) & 32767u];             // lane l -> bank l: one wavefront per load
        }
        idx += 512u;
    }
    if (acc == 0xFFFFFFFFu) out[0] = acc;
}

template <int KIND>   // 0 = LOP3/IADD3 (ALU pipe), 1 = IMAD (FMA pipe), 2 = both interleaved
__global__ void __launch_bounds__(kPeakThreads) peak_int_kernel(uint32_t* out, int iters, uint32_t m)
{
    uint32_t a[8], b[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = threadIdx.x + i; b[i] = blockIdx.x * 7u + i; }
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                // inline PTX so that the instruction mix is exactly what is counted (lop3 -> LOP3, mad.lo -> IMAD)
                if (KIND == 0) {
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x60;" : "+r"(a[i]) : "r"(b[i]), "r"(m));   // (a ^ b) & m
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(b[i]) : "r"(a[i]), "r"(m));   // b ^ a ^ m
                }
                if (KIND == 1) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(b[i]) : "r"(m), "r"(a[i]));
                if (KIND == 2) {
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x60;" : "+r"(a[i]) : "r"(b[i]), "r"(m));
                    asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(b[i]) : "r"(m), "r"(a[i]));
                }
            }
        }
    }
    uint32_t acc = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc += a[i] ^ b[i];
    if (acc == 0x12345u) out[0] = acc;
}

__global__ void __launch_bounds__(kPeakThreads) peak_fp64_kernel(double* out, int iters, double g)
{
    double a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = 1.0 + 1e-9 * (threadIdx.x + i);
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = __dadd_rn(__dmul_rn(a[i], g), 1.0e-3);  // DMUL + DADD, no FMA (as D6)
        }
    }
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc += a[i];
    if (acc == 12345.678) out[0] = acc;
}

__global__ void __launch_bounds__(kPeakThreads) peak_l2_kernel(const uint32_t* __restrict__ buf, uint32_t n_sectors_mask,
                                                               uint32_t* out, int iters)
{
    uint32_t x = (blockIdx.x * kPeakThreads + threadIdx.x) * 2654435761u + 99991u, acc = 0;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x = x * 1664525u + 1013904223u;
            acc += __ldcg(buf + (size_t)((x >> 8) & n_sectors_mask) * 8u);     // one word of a random 32-byte sector
        }
    }
    if (acc == 0xFFFFFFFFu) out[0] = acc;
}

template <typename F>
cudaError_t time_launch(F launch, cudaStream_t st, float* ms)
{
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    if ((e = cudaEventCreate(&e1)) != cudaSuccess) { cudaEventDestroy(e0); return e; }
    launch();                                                 // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {
        cudaEventRecord(e0, st);
        launch();
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        float t = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
        if (t < best) best = t;
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *ms = best;
    return e;
}

}  // namespace

cudaError_t measure_peaks(int n_sms, int clock_khz, double* out, cudaStream_t st, int64_t* n_launches)
{
    uint32_t* d_out = nullptr;
    uint32_t* d_buf = nullptr;
    const size_t l2_bytes = 64u << 20;
    cudaError_t e = cudaMalloc(&d_out, 64);
    if (e != cudaSuccess) return e;
    if ((e = cudaMalloc(&d_buf, l2_bytes)) != cudaSuccess) { cudaFree(d_out); return e; }
    cudaMemsetAsync(d_buf, 1, l2_bytes, st);
    const size_t smem = 128u * 1024u;
    cudaFuncSetAttribute(peak_lds_u8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(peak_lds_wave_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const int grid = n_sms, T = kPeakThreads;                 // one block per SM, 16 warps: the shape of mc_halo_kernel
    const double threads = (double)grid * T;
    float ms = 0.f;
    const int it_lds = 4000, it_int = 4000, it_f64 = 2000, it_l2 = 2000;
    if (e == cudaSuccess) e = time_launch([&] { peak_lds_u8_kernel<<<grid, T, smem, st>>>(d_out, it_lds); ++*n_launches; }, st, &ms);
    out[0] = threads * it_lds * 16.0 / (ms * 1e-3);
    if (e == cudaSuccess) e = time_launch([&] { peak_lds_wave_kernel<<<grid, T, smem, st>>>(d_out, it_lds); ++*n_launches; }, st, &ms);
    out[1] = threads / 32.0 * it_lds * 16.0 / (ms * 1e-3);
    if (e == cudaSuccess) e = time_launch([&] { peak_int_kernel<0><<<grid, T, 0, st>>>(d_out, it_int, 0x5bd1e995u); ++*n_launches; }, st, &ms);
    out[2] = threads * it_int * 4.0 * 8.0 * 2.0 / (ms * 1e-3);               // two LOP3 per element
    if (e == cudaSuccess) e = time_launch([&] { peak_int_kernel<1><<<grid, T, 0, st>>>(d_out, it_int, 0x5bd1e995u); ++*n_launches; }, st, &ms);
    out[3] = threads * it_int * 4.0 * 8.0 * 1.0 / (ms * 1e-3);
    if (e == cudaSuccess) e = time_launch([&] { peak_int_kernel<2><<<grid, T, 0, st>>>(d_out, it_int, 0x5bd1e995u); ++*n_launches; }, st, &ms);
    out[4] = threads * it_int * 4.0 * 8.0 * 2.0 / (ms * 1e-3);               // LOP3 + IMAD per element
    if (e == cudaSuccess) e = time_launch([&] { peak_fp64_kernel<<<grid, T, 0, st>>>(reinterpret_cast<double*>(d_out), it_f64, 0.999999); ++*n_launches; }, st, &ms);
    out[5] = threads * it_f64 * 4.0 * 8.0 * 2.0 / (ms * 1e-3);
    if (e == cudaSuccess)
        e = time_launch([&] { peak_l2_kernel<<<grid * 2, T, 0, st>>>(d_buf, (uint32_t)(l2_bytes / 32u - 1u), d_out, it_l2); ++*n_launches; }, st, &ms);
    out[6] = threads * 2.0 * it_l2 * 8.0 * 32.0 / (ms * 1e-3) / 1e9;
    out[7] = clock_khz / 1000.0;
    cudaFree(d_out);
    cudaFree(d_buf);
    return e;
}

}  // namespace hea
