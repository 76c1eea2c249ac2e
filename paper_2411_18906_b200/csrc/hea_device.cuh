// hea_device.cuh -- device-side parameter blocks and small helpers shared by the kernels of libhea_b200.
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cstring>
#include <cuda_runtime.h>

namespace hea {

constexpr int kSMM = 3 * 8 * 8;           // max S*M*M

// Constant tables of one context, resident in device global memory (copied to shared memory by the MC kernel).
struct DevTables {
    double g[kSMM];                       // g[s][i][j] = N / (z_s N_i N_j), compact index (s*M + i)*M + j  (D5-D6)
    double t[kSMM];                       // alpha target, same index
    double w[4];                          // shell weights
    int8_t stencil[4 * 42 * 4];           // [b][e] -> (nb, sx, sy, sz), e over the concatenated shells, stride Z
    uint8_t by_basis[4 * 42];             // [b][i], stride Z: the entry that comes i-th when every shell's entries are
                                          // ordered by the neighbour's basis index nb (stable); stays within the shell
};

// Scalars passed by value to every kernel.
struct KParams {
    int N;                                // sites
    int Npad;                             // N rounded up to a multiple of 32: rows of the table (whole 32-site tiles)
    int M, S, Z, A;
    int L[3];
    int z[3];
    int zoff[4];
    int m_self[3];                        // per shell: table entries of a site that are the site itself (0 unless a tiny cell)
    const int32_t* nbr_site;              // [Npad][Z] site-major: the Z neighbours of one site are contiguous
    const DevTables* tab;
};

// ---------------------------------------------------------------- Philox4x32-10 (Salmon et al. SC'11; D7)
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1)
{
    constexpr uint32_t MUL_A = 0xD2511F53u, MUL_B = 0xCD9E8D57u;
    constexpr uint32_t BUMP_A = 0x9E3779B9u, BUMP_B = 0xBB67AE85u;
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t a_hi = __umulhi(MUL_A, c0), a_lo = MUL_A * c0;
        const uint32_t b_hi = __umulhi(MUL_B, c2), b_lo = MUL_B * c2;
        c0 = b_hi ^ c1 ^ k0;
        c1 = b_lo;
        c2 = a_hi ^ c3 ^ k1;
        c3 = a_lo;
        k0 += BUMP_A;
        k1 += BUMP_B;
    }
    return make_uint4(c0, c1, c2, c3);
}

// The same generator with the ten round keys precomputed (rk[2r], rk[2r+1] = key + r * bump): when rk lives in
// kernel-parameter space the keys are constant-bank operands of the xors and cost no instruction.
__device__ __forceinline__ uint4 philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const uint32_t (&rk)[20])
{
    constexpr uint32_t MUL_A = 0xD2511F53u, MUL_B = 0xCD9E8D57u;
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t a_hi = __umulhi(MUL_A, c0), a_lo = MUL_A * c0;
        const uint32_t b_hi = __umulhi(MUL_B, c2), b_lo = MUL_B * c2;
        c0 = b_hi ^ c1 ^ rk[2 * round];
        c1 = b_lo;
        c2 = a_hi ^ c3 ^ rk[2 * round + 1];
        c3 = a_lo;
    }
    return make_uint4(c0, c1, c2, c3);
}

// Exact int32 -> double without the conversion (XU) pipe: 2^52 + 2^31 + n is exactly representable, so the mantissa
// can be written directly and the constant subtracted exactly.  Bit-identical to (double)n for every int32.
__device__ __forceinline__ double i2d_exact(int n)
{
    return __dsub_rn(__hiloint2double(0x43300000, (int)((unsigned)n ^ 0x80000000u)), 4503601774854144.0);
}

// Order-preserving map of a double onto unsigned 64-bit integers (x < y  <=>  key(x) < key(y), also for negative values:
// J can be negative when a shell weight is).  -0.0 sorts below +0.0; J is a sum started from +0.0 and never is -0.0.
__host__ __device__ __forceinline__ unsigned long long ordered_bits(double x)
{
#ifdef __CUDA_ARCH__
    const unsigned long long b = (unsigned long long)__double_as_longlong(x);
#else
    unsigned long long b;
    memcpy(&b, &x, sizeof b);
#endif
    return b ^ ((b >> 63) ? ~0ull : (1ull << 63));
}

// D6: one squared deviation, every operation individually rounded (no FMA contraction).
__device__ __forceinline__ double sq_dev(int n, double g, double t)
{
    const double x = __dmul_rn(i2d_exact(n), g);
    const double al = __dsub_rn(1.0, x);
    const double d = __dsub_rn(al, t);
    return __dmul_rn(d, d);
}

}  // namespace hea
