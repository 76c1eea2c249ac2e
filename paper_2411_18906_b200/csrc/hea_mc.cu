// hea_mc.cu -- chain-parallel Monte Carlo local search (hea_mc_run).
// DESIGN.md D6, D7, D9; Alg. 3, Eq. 4, Eq. 5, Eq. 6.
//
// One persistent launch runs all n_steps steps; no host round trip inside.  One thread block per chain.
//   - the chain's configuration lives in shared memory (uint8, or 4-bit packed when that is what fits), else it is
//     read through L1/L2 from global memory; counts, g, t, w live in shared memory;
//   - a GROUP of G lanes (G = 1..32, a power of two) owns one candidate: all lanes derive the same Philox block
//     (counter = step, k, chain), then split the 2Z neighbour entries of the two sites between them; each lane
//     accumulates sum_{nbrs of b} e_r - sum_{nbrs of a} e_r as one packed 64-bit word per shell (8-bit fields,
//     wrap-around arithmetic; a bias makes the fields non-negative after the group reduction by shuffles);
//   - the S*M rows of the objective are split between the lanes of the group, then combined by shuffles in the
//     fixed D6 order (rows i ascending within a shell, shells ascending), every operation individually rounded;
//   - improving candidates post their index with a shared-memory atomicMin (triple-buffered so that a step without
//     an accepted move needs ONE block barrier); the owning group applies the move.
// Results are a function of (seed, chain, step) only: independent of G, block size and occupancy placement.
#include "hea_device.cuh"

namespace hea {

namespace {

enum { OCC_SMEM_U8 = 1, OCC_SMEM_NIB = 2, OCC_GLOBAL = 3 };

constexpr uint64_t kBias = 0x8080808080808080ULL;
constexpr int kNoCandidate = 0x7FFFFFFF;

template <int OCC>
struct OccView {
    uint8_t* p;
    __device__ __forceinline__ uint32_t get(uint32_t i) const
    {
        if (OCC == OCC_SMEM_NIB) return (p[i >> 1] >> ((i & 1u) * 4u)) & 0xFu;
        return p[i];
    }
    __device__ __forceinline__ void set(uint32_t i, uint32_t v) const
    {
        if (OCC == OCC_SMEM_NIB) {
            const uint32_t sh = (i & 1u) * 4u;
            p[i >> 1] = (uint8_t)((p[i >> 1] & ~(0xFu << sh)) | (v << sh));
        } else {
            p[i] = (uint8_t)v;
        }
    }
};

struct ChainShared {
    double g[kSMM];
    double t[kSMM];
    double w[4];
    int cnt[kSMM];
    double J;
    unsigned long long n_accept, n_null, hash, last_accept, n_logged;
    int best[3];
    int pad;
};

__device__ __forceinline__ int field8(uint64_t packed, int r) { return (int)((packed >> (8 * r)) & 0xFFu) - 128; }

// dN[s][i][j] for a swap of species p (site a) and q (site b), given the biased packed word of shell s whose
// field r is  #(nbrs of b with species r) - #(nbrs of a with species r)  (a, b themselves excluded):
//   N[p][r] += d[r]; N[r][p] += d[r]; N[q][r] -= d[r]; N[r][q] -= d[r]
__device__ __forceinline__ int delta_cell(uint64_t packed, int i, int j, int p, int q)
{
    const int ci = (i == p) - (i == q);
    const int cj = (j == p) - (j == q);
    return ci * field8(packed, j) + cj * field8(packed, i);
}

template <int G, int OCC>
__global__ void __launch_bounds__(1024)
mc_chain_kernel(const KParams P, uint8_t* __restrict__ occ_all, int32_t* __restrict__ counts_all,
                unsigned long long n_steps, int K, unsigned long long seed, unsigned long long chain0,
                unsigned long long step0, unsigned long long* __restrict__ stats_all,
                unsigned long long* __restrict__ log_all, long long log_cap)
{
    extern __shared__ __align__(16) uint8_t s_raw[];
    ChainShared& sh = *reinterpret_cast<ChainShared*>(s_raw);
    uint8_t* s_occ = s_raw + sizeof(ChainShared);

    const int tid = threadIdx.x, T = blockDim.x;
    const int M = P.M, S = P.S, Z = P.Z, N = P.N;
    const int SM = S * M, SMM = SM * M;
    const size_t chain_local = blockIdx.x;
    uint8_t* g_occ = occ_all + chain_local * (size_t)N;
    int32_t* g_cnt = counts_all + chain_local * (size_t)SMM;
    unsigned long long* g_stats = stats_all + chain_local * 5;
    const uint32_t chain = (uint32_t)(chain0 + chain_local);
    const uint32_t key0 = (uint32_t)seed, key1 = (uint32_t)(seed >> 32);

    // ---- prologue: constants, counts, configuration -> shared memory
    for (int i = tid; i < SMM; i += T) { sh.g[i] = P.tab->g[i]; sh.t[i] = P.tab->t[i]; sh.cnt[i] = g_cnt[i]; }
    if (tid < 4) sh.w[tid] = P.tab->w[tid];
    if (OCC == OCC_SMEM_U8) {
        for (int i = tid; i < N; i += T) s_occ[i] = g_occ[i];
    } else if (OCC == OCC_SMEM_NIB) {
        for (int i = tid; i < (N + 1) / 2; i += T) {
            const uint32_t lo = g_occ[2 * i], hi = (2 * i + 1 < N) ? g_occ[2 * i + 1] : 0u;
            s_occ[i] = (uint8_t)(lo | (hi << 4));
        }
    }
    if (tid == 0) {
        sh.n_accept = g_stats[0]; sh.n_null = 0; sh.hash = g_stats[2]; sh.last_accept = g_stats[3]; sh.n_logged = 0;
        sh.best[0] = sh.best[1] = sh.best[2] = kNoCandidate;
    }
    __syncthreads();
    if (tid == 0) {       // J of the supplied counts, D6 order
        double J = 0.0;
        for (int s = 0; s < S; ++s) {
            double shs = 0.0;
            for (int i = 0; i < M; ++i) {
                double row = 0.0;
                for (int j = 0; j < M; ++j) {
                    const int idx = (s * M + i) * M + j;
                    row = __dadd_rn(row, sq_dev(sh.cnt[idx], sh.g[idx], sh.t[idx]));
                }
                shs = __dadd_rn(shs, row);
            }
            J = __dadd_rn(J, __dmul_rn(sh.w[s], shs));
        }
        sh.J = J;
    }
    __syncthreads();

    const OccView<OCC> occ{OCC == OCC_GLOBAL ? g_occ : s_occ};
    const int gl = tid & (G - 1);                 // lane within the group
    // shuffle mask = the lanes of this group (groups of one warp may be at different candidates)
    const uint32_t gmask = G == 32 ? 0xFFFFFFFFu : (((1u << G) - 1u) << ((tid & 31) & ~(G - 1)));
    const int group = tid / G, n_groups = T / G;
    const int z1 = P.zoff[1], z2 = P.zoff[2];
    const int32_t* __restrict__ nbr = P.nbr_site;
    unsigned int my_null = 0;

    for (unsigned long long it = 0; it < n_steps; ++it) {
        const unsigned long long step = step0 + it;
        const int buf = (int)(it % 3);
        const double J_cur = sh.J;
        // first improving candidate of this group (k ascending within the group's loop)
        int win_k = kNoCandidate;
        uint32_t win_a = 0, win_b = 0, win_p = 0, win_q = 0;
        uint64_t win_d0 = 0, win_d1 = 0, win_d2 = 0;
        double win_J = 0.0;

        for (int k = group; k < K; k += n_groups) {
            // ---- D9.1 proposal
            const uint4 r = philox4x32_10((uint32_t)step, (uint32_t)(step >> 32), (uint32_t)k, chain, key0, key1);
            uint32_t a = __umulhi(r.x, (uint32_t)N), b = __umulhi(r.y, (uint32_t)N - 1u);
            b += (b >= a);
            uint32_t p = occ.get(a), q = occ.get(b);
            if (p == q) {
                a = __umulhi(r.z, (uint32_t)N); b = __umulhi(r.w, (uint32_t)N - 1u);
                b += (b >= a);
                p = occ.get(a); q = occ.get(b);
                if (p == q) { my_null += (gl == 0); continue; }
            }
            // ---- D9.2 integer delta: packed per-shell  sum_b - sum_a  over this lane's share of the 2Z entries
            uint64_t d0 = 0, d1 = 0, d2 = 0;
            for (int e = gl; e < 2 * Z; e += G) {
                const bool second = e >= Z;
                const int ee = second ? e - Z : e;
                const uint32_t u = second ? b : a;
                const uint32_t v = (uint32_t)__ldg(nbr + (size_t)u * Z + ee);
                if (v != a && v != b) {
                    const uint64_t one = 1ull << (8 * occ.get(v));
                    const uint64_t val = second ? one : (0ull - one);
                    if (ee < z1) d0 += val; else if (ee < z2) d1 += val; else d2 += val;
                }
            }
            if (G > 1) {
#pragma unroll
                for (int off = G / 2; off >= 1; off >>= 1) {
                    d0 += __shfl_xor_sync(gmask, d0, off, G);
                    d1 += __shfl_xor_sync(gmask, d1, off, G);
                    if (S > 2) d2 += __shfl_xor_sync(gmask, d2, off, G);
                }
            }
            d0 += kBias; d1 += kBias; d2 += kBias;
            // ---- D6 objective from counts + delta: rows split over the lanes, combined in fixed order
            double Jk = 0.0, shell_sum = 0.0;
            for (int base = 0; base < SM; base += G) {
                const int row = base + gl;
                double row_sum = 0.0;
                if (row < SM) {
                    const int s = row / M, i = row - s * M;
                    const uint64_t d = s == 0 ? d0 : (s == 1 ? d1 : d2);
                    const int idx0 = row * M;
                    for (int j = 0; j < M; ++j) {
                        const int n = sh.cnt[idx0 + j] + delta_cell(d, i, j, (int)p, (int)q);
                        row_sum = __dadd_rn(row_sum, sq_dev(n, sh.g[idx0 + j], sh.t[idx0 + j]));
                    }
                }
#pragma unroll
                for (int l = 0; l < G; ++l) {
                    const int rr = base + l;
                    const double v = G > 1 ? __shfl_sync(gmask, row_sum, l, G) : row_sum;
                    if (rr < SM) {
                        shell_sum = __dadd_rn(shell_sum, v);
                        const int s = rr / M;
                        if (rr - s * M == M - 1) {
                            Jk = __dadd_rn(Jk, __dmul_rn(sh.w[s], shell_sum));
                            shell_sum = 0.0;
                        }
                    }
                }
            }
            if (Jk < J_cur && win_k == kNoCandidate) {
                win_k = k; win_a = a; win_b = b; win_p = p; win_q = q;
                win_d0 = d0; win_d1 = d1; win_d2 = d2; win_J = Jk;
                if (gl == 0) atomicMin(&sh.best[buf], k);
            }
        }
        __syncthreads();                                   // B1: all candidates evaluated, minimum posted
        const int k_best = sh.best[buf];
        if (tid == 0) sh.best[(buf + 2) % 3] = kNoCandidate;   // next user of that slot is two barriers away
        if (k_best != kNoCandidate) {
            if (win_k == k_best) {                         // the owning group applies the move (D9.4)
                for (int idx = gl; idx < SMM; idx += G) {
                    const int s = idx / (M * M), rem = idx - s * M * M, i = rem / M, j = rem - i * M;
                    const uint64_t d = s == 0 ? win_d0 : (s == 1 ? win_d1 : win_d2);
                    sh.cnt[idx] += delta_cell(d, i, j, (int)win_p, (int)win_q);
                }
                if (gl == 0) {
                    occ.set(win_a, win_q);
                    occ.set(win_b, win_p);
                    sh.J = win_J;
                    sh.n_accept += 1;
                    sh.last_accept = step;
                    unsigned long long h = sh.hash;
                    h = (h ^ (uint32_t)step) * 0x100000001b3ULL;
                    h = (h ^ (uint32_t)(step >> 32)) * 0x100000001b3ULL;
                    h = (h ^ (uint32_t)k_best) * 0x100000001b3ULL;
                    h = (h ^ win_a) * 0x100000001b3ULL;
                    h = (h ^ win_b) * 0x100000001b3ULL;
                    sh.hash = h;
                    const unsigned long long nl = sh.n_logged;
                    if (log_all != nullptr && (long long)nl < log_cap) {
                        unsigned long long* rec = log_all + (chain_local * (size_t)log_cap + nl) * 3;
                        rec[0] = step;
                        rec[1] = (unsigned long long)(uint32_t)k_best | ((unsigned long long)win_a << 32);
                        rec[2] = (unsigned long long)win_b;
                    }
                    sh.n_logged = nl + 1;
                }
            }
            __syncthreads();                               // B2: the move is visible before the next step's reads
        }
    }

    // ---- epilogue: write back
    if (my_null) atomicAdd(&sh.n_null, (unsigned long long)my_null);
    __syncthreads();
    if (OCC == OCC_SMEM_U8) {
        for (int i = tid; i < N; i += T) g_occ[i] = s_occ[i];
    } else if (OCC == OCC_SMEM_NIB) {
        for (int i = tid; i < N; i += T) g_occ[i] = (uint8_t)occ.get(i);
    }
    for (int i = tid; i < SMM; i += T) g_cnt[i] = sh.cnt[i];
    if (tid == 0) {
        g_stats[0] = sh.n_accept;
        g_stats[1] += sh.n_null;
        g_stats[2] = sh.hash;
        g_stats[3] = sh.last_accept;
        g_stats[4] = (unsigned long long)__double_as_longlong(sh.J);
    }
}

template <int G, int OCC>
cudaError_t launch_one(const KParams& P, uint8_t* occ, int32_t* counts, int64_t C, uint64_t n_steps, int K,
                       uint64_t seed, uint64_t chain0, uint64_t step0, void* stats, void* log, int64_t log_cap,
                       int threads, size_t smem, cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(mc_chain_kernel<G, OCC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    mc_chain_kernel<G, OCC><<<(unsigned)C, threads, smem, st>>>(
        P, occ, counts, (unsigned long long)n_steps, K, (unsigned long long)seed, (unsigned long long)chain0,
        (unsigned long long)step0, reinterpret_cast<unsigned long long*>(stats),
        reinterpret_cast<unsigned long long*>(log), (long long)log_cap);
    return cudaGetLastError();
}

template <int G>
cudaError_t launch_occ(int occ_mode, const KParams& P, uint8_t* occ, int32_t* counts, int64_t C, uint64_t n_steps,
                       int K, uint64_t seed, uint64_t chain0, uint64_t step0, void* stats, void* log,
                       int64_t log_cap, int threads, size_t smem, cudaStream_t st)
{
    switch (occ_mode) {
        case OCC_SMEM_U8:
            return launch_one<G, OCC_SMEM_U8>(P, occ, counts, C, n_steps, K, seed, chain0, step0, stats, log, log_cap, threads, smem, st);
        case OCC_SMEM_NIB:
            return launch_one<G, OCC_SMEM_NIB>(P, occ, counts, C, n_steps, K, seed, chain0, step0, stats, log, log_cap, threads, smem, st);
        default:
            return launch_one<G, OCC_GLOBAL>(P, occ, counts, C, n_steps, K, seed, chain0, step0, stats, log, log_cap, threads, smem, st);
    }
}

}  // namespace

size_t mc_shared_bytes(int occ_mode, int N)
{
    size_t s = sizeof(ChainShared);
    if (occ_mode == OCC_SMEM_U8) s += (size_t)N;
    else if (occ_mode == OCC_SMEM_NIB) s += (size_t)(N + 1) / 2;
    return (s + 15) & ~(size_t)15;
}

cudaError_t launch_mc(const KParams& P, int lanes, int occ_mode, int threads, uint8_t* occ, int32_t* counts,
                      int64_t C, uint64_t n_steps, int K, uint64_t seed, uint64_t chain0, uint64_t step0,
                      void* stats, void* log, int64_t log_cap, cudaStream_t st, int64_t* n_launches)
{
    const size_t smem = mc_shared_bytes(occ_mode, P.N);
    cudaError_t e;
#define HEA_MC_CASE(GG) \
    case GG: e = launch_occ<GG>(occ_mode, P, occ, counts, C, n_steps, K, seed, chain0, step0, stats, log, log_cap, threads, smem, st); break;
    switch (lanes) {
        HEA_MC_CASE(1)
        HEA_MC_CASE(2)
        HEA_MC_CASE(4)
        HEA_MC_CASE(8)
        HEA_MC_CASE(16)
        default: e = launch_occ<32>(occ_mode, P, occ, counts, C, n_steps, K, seed, chain0, step0, stats, log, log_cap, threads, smem, st); break;
    }
#undef HEA_MC_CASE
    if (e == cudaSuccess) ++*n_launches;
    return e;
}

}  // namespace hea
