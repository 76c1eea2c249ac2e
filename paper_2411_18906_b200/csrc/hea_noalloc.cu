// hea_noalloc.cu -- hea_pool_rank_static: the ranking step of hea_pool_select (Alg. 1, P:178-195, P:207;
// DESIGN.md A24) for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc).  Product code (sm_100a); nothing from oracle/.
//
// hea_pool_select keeps the J of every chain in a context-owned scratch buffer that grows by cudaMalloc.  Here the same
// scratch is a file-scope `static __device__` array of a fixed, stated size (kPoolRankStaticMax chains x 8 bytes =
// 512 KB): every GPU that loads the library holds it until the process exits.  Nothing on this path calls cudaMalloc,
// cudaFree or an allocating library routine.
//
// In HOST code the array's name is only a host-side stand-in for the symbol, never a device address, so the launcher
// resolves the address with cudaGetSymbolAddress -- once per device, with that device current -- and hands the
// resolved pointer to the kernels.
//
// The array is shared by every call in the process and keeps the last call's contents.  Nothing in it has to start at
// zero: the objective kernel overwrites entries [0, C) before the ranking kernel reads exactly those entries, on the same
// stream.  Calls that overlap on one GPU (two streams, two contexts, two threads) race on it: serialise them.
#include <cstdint>
#include <mutex>
#include <string>
#include <cuda_runtime.h>

#include "hea_device.cuh"

namespace hea {

// hea_sro.cu: J of each configuration from its counts, D6 order (the launcher hea_pool_select uses as well)
cudaError_t launch_sro_epilogue(const KParams& P, const int32_t* counts, int64_t B, double* alpha, double* obj,
                                cudaStream_t st, int64_t* n_launches);

constexpr int64_t kPoolRankStaticMax = 65536;          // == HEA_POOL_RANK_STATIC_MAX of include/hea.h
constexpr int kMaxDevices = 64;

namespace {

// The scratch: J of chain c at [c].  512 KB per GPU, for the life of the process.
static __device__ __align__(256) double g_pool_rank_J[kPoolRankStaticMax];

std::mutex g_mu;
double* g_J_ptr[kMaxDevices] = {nullptr};               // resolved device address of g_pool_rank_J, per device ordinal

// order[r] = index of the chain of rank r (J ascending, ties -> lower index), for r < n_keep: pool_rank_kernel of
// hea_pool.cu with a block's slice of the keys staged in shared memory, J read from the static scratch.
constexpr int kRankThreads = 256;

__global__ void __launch_bounds__(kRankThreads) pool_rank_static_kernel(const double* __restrict__ J, int64_t C, int64_t n_keep,
                                                                        int32_t* __restrict__ order)
{
    __shared__ unsigned long long s_key[kRankThreads];
    const int64_t c = (int64_t)blockIdx.x * kRankThreads + threadIdx.x;
    const unsigned long long mine = c < C ? ordered_bits(J[c]) : ~0ull;
    int64_t rank = 0;
    for (int64_t o0 = 0; o0 < C; o0 += kRankThreads) {
        const int64_t o = o0 + threadIdx.x;
        __syncthreads();
        s_key[threadIdx.x] = o < C ? ordered_bits(J[o]) : ~0ull;
        __syncthreads();
        const int n = (int)((C - o0) < kRankThreads ? (C - o0) : kRankThreads);
        for (int i = 0; i < n; ++i) {
            const unsigned long long other = s_key[i];
            rank += (other < mine) || (other == mine && o0 + i < c);
        }
    }
    if (c < C && rank < n_keep) order[rank] = (int32_t)c;
}

// Device address of the static scratch on `device` (which must be the current device).  Resolved once per device.
cudaError_t static_scratch(int device, double** out, std::string* err)
{
    if (device < 0 || device >= kMaxDevices) {
        *err = "device ordinal beyond the " + std::to_string(kMaxDevices) + " this entry point keeps an address for";
        return cudaErrorInvalidDevice;
    }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_J_ptr[device]) {
        double* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_pool_rank_J);
        if (e != cudaSuccess || !p) {
            (void)cudaGetLastError();
            *err = std::string("cudaGetSymbolAddress(static scratch): ") + cudaGetErrorString(e);
            return e != cudaSuccess ? e : cudaErrorInvalidSymbol;
        }
        g_J_ptr[device] = p;
    }
    *out = g_J_ptr[device];
    return cudaSuccess;
}

}  // namespace

// `device` is the current device (the caller holds a device guard).  C in [1, kPoolRankStaticMax], 0 <= n_keep <= C.
cudaError_t pool_rank_static(const KParams& P, int device, const int32_t* counts, int64_t C, int64_t n_keep, int32_t* order,
                             cudaStream_t st, int64_t* n_launches, std::string* err)
{
    if (C < 1 || C > kPoolRankStaticMax) {
        *err = "C is beyond the static scratch";
        return cudaErrorInvalidValue;
    }
    double* J = nullptr;
    cudaError_t e = static_scratch(device, &J, err);
    if (e != cudaSuccess) return e;
    e = launch_sro_epilogue(P, counts, C, nullptr, J, st, n_launches);               // J[0..C) overwritten
    if (e != cudaSuccess) { *err = std::string("objective kernel: ") + cudaGetErrorString(e); return e; }
    pool_rank_static_kernel<<<(unsigned)((C + kRankThreads - 1) / kRankThreads), kRankThreads, 0, st>>>(J, C, n_keep, order);
    ++*n_launches;
    e = cudaGetLastError();
    if (e != cudaSuccess) *err = std::string("ranking kernel: ") + cudaGetErrorString(e);
    return e;
}

}  // namespace hea
