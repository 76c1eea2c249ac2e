// hea_mc_common.cuh -- pieces shared by the Monte Carlo kernels of libhea_b200 (hea_mc.cu, hea_mc2.cu): move records,
// kernel arguments, the packed per-shell histogram difference and the D6 shell sum.  Product code; nothing from oracle/.
#pragma once
#include <cstdint>
#include <type_traits>

#include "hea_device.cuh"

namespace hea {

constexpr uint32_t kNoKey = 0xFFFFFFFFu;     // "no improving candidate"; real keys are (window step << 10) | k
constexpr int kMaxCluster = 8;
constexpr int kMaxRounds = 8;                // candidates per thread per window when W > 1

// The best move of one block in one window, posted to every replica.
struct MoveRec {
    uint32_t key;                 // (window step << 10) | k, kNoKey if none
    uint32_t a, b, pq;            // sites; species p | q << 8
    double J;
    uint64_t d[3];                // packed neighbour-histogram differences per shell (Pack<M>::W, biased fields)
};

struct ChainShared {
    int cnt[kSMM];
    double J;
    unsigned long long n_accept, n_null, hash, last_accept, n_logged;
    uint32_t best[3];             // local minimum key, triple-buffered (one block barrier per window)
    uint32_t pad;
    MoveRec rec[2][kMaxCluster];  // [window parity][source block]
};

// Objective constants in kernel-parameter (constant-bank) space: operands of the fp64 instructions, no loads.
template <int M>
struct McConst {
    double g[3 * M * M];
    double t[3 * M * M];
    double w[4];
};

struct McArgs {
    uint8_t* occ_all;
    int32_t* counts_all;
    unsigned long long n_steps, seed, chain0, step0;
    unsigned long long* stats_all;
    unsigned long long* log_all;
    long long log_cap;
    int K;
    int R;                        // blocks per chain (cluster size)
    int w_max;                    // cap on the window length in steps (>= 1)
    int fast_nbr;                 // 1: interior sites take neighbours as site + offset (shared-memory stencil), no table load
    int prune;                    // 1: all shell weights >= 0, so every shell term w_s*sh_s is an exact lower bound of J (see below)
};

// Packed per-shell histogram difference: one signed field per species, value in [-24, 24] (a shell has <= 24
// neighbours), stored biased so that the fields never borrow from each other after the final add of the bias.
//   M <= 4: 8-bit fields in 32 bits;  M == 5: 6-bit fields in 32 bits (30 used);  M >= 6: 8-bit fields in 64 bits.
template <int M>
struct Pack {
    static constexpr int FB = (M == 5) ? 6 : 8;
    static constexpr bool k32 = M * FB <= 32;
    using W = typename std::conditional<k32, uint32_t, uint64_t>::type;
    static constexpr int kHalf = 1 << (FB - 1);
    __host__ __device__ static constexpr W bias()
    {
        W b = 0;
        for (int r = 0; r < M; ++r) b |= (W)kHalf << (FB * r);
        return b;
    }
    __device__ __forceinline__ static W one(uint32_t species) { return (W)1 << (FB * species); }
    __device__ __forceinline__ static int field(W packed, int r) { return (int)((packed >> (FB * r)) & (W)((1 << FB) - 1)) - kHalf; }
};

// One shell's contribution  sum_i sum_j (1 - (N_ij + dN_ij) g_ij - t_ij)^2  in the D6 order.
// dN[i][j] = ci*F[j] + cj*F[i], ci = [i==p] - [i==q], F[r] = #(nbrs of b of species r) - #(nbrs of a ...) (a, b excluded).
// SYM: target symmetric (t_ij == t_ji bitwise; g and the counts of a recount always are), so e_ji is the same sequence of
// operations on the same operands as e_ij and is reused instead of recomputed; the additions keep the D6 order.
template <int M, bool SYM>
__device__ __forceinline__ double shell_sum(const int* __restrict__ cnt, const double* __restrict__ g,
                                            const double* __restrict__ t, typename Pack<M>::W dpacked, int p, int q)
{
    int F[M], c[M];
#pragma unroll
    for (int r = 0; r < M; ++r) { F[r] = Pack<M>::field(dpacked, r); c[r] = (r == p) - (r == q); }
    double up[M * M];               // only entries (i, j > i) are live when SYM
    double sh = 0.0;
#pragma unroll
    for (int i = 0; i < M; ++i) {
        double row = 0.0;
#pragma unroll
        for (int j = 0; j < M; ++j) {
            double e;
            if (SYM && j < i) {
                e = up[j * M + i];
            } else {
                const int n = cnt[i * M + j] + c[i] * F[j] + c[j] * F[i];
                e = sq_dev(n, g[i * M + j], t[i * M + j]);
                if (SYM && j > i) up[i * M + j] = e;
            }
            row = __dadd_rn(row, e);
        }
        sh = __dadd_rn(sh, row);
    }
    return sh;
}

}  // namespace hea
