// hea_pool.cu -- selection step of the global search (hea_pool_select): rank the chains of a pool by J and move the best
// to the front.  PAPER.md Alg. 1; A24.  Product code (sm_100a); nothing from oracle/.
#include <cstdint>
#include <cuda_runtime.h>

#include "hea_device.cuh"

namespace hea {

namespace {

// order[r] = index of the chain of rank r (J ascending, ties -> lower index), for r < n_keep.  J is compared through the
// order-preserving integer key of hea_device.cuh (negative J, possible with a negative shell weight, included).
// One thread per chain, O(C^2) compares over an L2-resident array: C <= 65,536.
__global__ void pool_rank_kernel(const double* __restrict__ J, int64_t C, int64_t n_keep, int32_t* __restrict__ order)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= C) return;
    const unsigned long long mine = ordered_bits(J[c]);
    int64_t rank = 0;
    for (int64_t o = 0; o < C; ++o) {
        const unsigned long long other = ordered_bits(__ldg(J + o));
        rank += (other < mine) || (other == mine && o < c);
    }
    if (rank < n_keep) order[rank] = (int32_t)c;
}

// dst[r][0..item) = src[order[r]][0..item), bytes; grid (chunks, n_keep)
__global__ void pool_gather_kernel(const uint8_t* __restrict__ src, uint8_t* __restrict__ dst,
                                   const int32_t* __restrict__ order, size_t item)
{
    const uint8_t* s = src + (size_t)order[blockIdx.y] * item;
    uint8_t* d = dst + (size_t)blockIdx.y * item;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < item; i += (size_t)gridDim.x * blockDim.x) d[i] = s[i];
}

}  // namespace

cudaError_t launch_pool_rank(const double* J, int64_t C, int64_t n_keep, int32_t* order, cudaStream_t st, int64_t* n_launches)
{
    pool_rank_kernel<<<(unsigned)((C + 255) / 256), 256, 0, st>>>(J, C, n_keep, order);
    ++*n_launches;
    return cudaGetLastError();
}

cudaError_t launch_pool_gather(const void* src, void* dst, const int32_t* order, int64_t n_keep, size_t item,
                               cudaStream_t st, int64_t* n_launches)
{
    if (n_keep == 0 || item == 0) return cudaSuccess;
    for (int64_t r0 = 0; r0 < n_keep; r0 += 65535) {
        const unsigned ny = (unsigned)((n_keep - r0) < 65535 ? (n_keep - r0) : 65535);
        const unsigned nx = (unsigned)((item + 256 * 16 - 1) / (256 * 16) < 1 ? 1 : (item + 256 * 16 - 1) / (256 * 16));
        pool_gather_kernel<<<dim3(nx, ny), 256, 0, st>>>(reinterpret_cast<const uint8_t*>(src),
                                                        reinterpret_cast<uint8_t*>(dst) + (size_t)r0 * item, order + r0, item);
        ++*n_launches;
    }
    return cudaGetLastError();
}

}  // namespace hea
