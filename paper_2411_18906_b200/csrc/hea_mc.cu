// hea_mc.cu -- chain-parallel Monte Carlo local search (hea_mc_run).
// DESIGN.md D6, D7, D9 and section 5; Alg. 3, Eq. 4, Eq. 5, Eq. 6.
//
// One persistent launch runs all n_steps steps of every chain; no host round trip inside.
//
// Mapping.  A chain is owned by one thread block, or by a thread-block CLUSTER of R blocks (R = 2, 4, 8) when there
// are fewer chains than SMs; every block of a cluster keeps its own replica of the chain state (occupancy, pair
// counts, J) in shared memory and all replicas apply the same moves.  One THREAD evaluates one candidate swap:
// Philox block -> sites (a, b) -> species histograms of the neighbours of a and b as one packed word per shell
// (8-bit fields, wrap-around arithmetic) -> J from counts + delta in the fixed D6 order (fp64, no FMA).
//
// Speculative step windows.  The steps of a chain depend on each other only through accepted moves, and D9 applies
// the lowest-index improving candidate.  So a WINDOW of W consecutive steps (W*K candidates, ordered by (step, k))
// is evaluated against the same configuration; the lowest improving (step, k) in the window is exactly the move D9
// would apply first; it is applied, the steps after it are discarded and the next window starts at step + 1.
// Without an accepted move the whole window is committed.  W adapts (doubles after a window without a move, falls
// back to the observed gap after one), so the converged "reject regime" fills the machine while the early "accept
// regime" wastes little.  The trajectory is identical to the step-by-step definition for every W, R and block size.
//
// Per window: one block barrier (+ one cluster barrier when R > 1: every block posts its local best move record into
// every peer's shared memory through DSMEM, then all replicas apply the global minimum).
#include <cooperative_groups.h>

#include <cstring>
#include <type_traits>

#include "hea_device.cuh"
#include "hea_mc_common.cuh"

namespace cg = cooperative_groups;

namespace hea {

namespace {

enum { OCC_SMEM_U8 = 1, OCC_SMEM_NIB = 2, OCC_GLOBAL = 3 };

template <int OCC>
struct OccView {
    uint8_t* p;
    __device__ __forceinline__ uint32_t get(uint32_t i) const
    {
        if (OCC == OCC_SMEM_NIB) return (p[i >> 1] >> ((i & 1u) * 4u)) & 0xFu;
        if (OCC == OCC_GLOBAL) return __ldcg(p + i);       // L2: coherent across the blocks of a cluster
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

template <int M, int OCC, bool SYM>
__global__ void __launch_bounds__(1024)
mc_window_kernel(const KParams P, const __grid_constant__ McConst<M> Kc, const McArgs A)
{
    extern __shared__ __align__(16) uint8_t s_raw[];
    ChainShared& sh = *reinterpret_cast<ChainShared*>(s_raw);
    // shared layout: ChainShared | neighbour index offsets [A][Z] | interior-site bitmap [ceil(N/32)] | occupancy
    int* s_ds = reinterpret_cast<int*>(s_raw + sizeof(ChainShared));
    uint32_t* s_bm = reinterpret_cast<uint32_t*>(s_ds + ((P.A * P.Z + 3) & ~3));
    const bool FAST = OCC != OCC_GLOBAL && A.fast_nbr != 0;
    uint8_t* s_occ = reinterpret_cast<uint8_t*>(s_bm + (FAST ? ((P.N + 127) >> 7) << 2 : 0));

    const int tid = threadIdx.x, T = blockDim.x;
    const int S = P.S, Z = P.Z, N = P.N, K = A.K, R = A.R;
    constexpr int MM = M * M;
    using PW = typename Pack<M>::W;
    const int SMM = S * MM;
    const uint32_t rank = R > 1 ? cg::this_cluster().block_rank() : 0u;
    const size_t chain_local = blockIdx.x / (unsigned)R;
    uint8_t* g_occ = A.occ_all + chain_local * (size_t)N;
    int32_t* g_cnt = A.counts_all + chain_local * (size_t)SMM;
    unsigned long long* g_stats = A.stats_all + chain_local * 5;
    const uint32_t chain = (uint32_t)(A.chain0 + chain_local);
    const uint32_t key0 = (uint32_t)A.seed, key1 = (uint32_t)(A.seed >> 32);

    // ---- prologue: counts, configuration -> shared memory; J of the supplied counts (D6 order)
    for (int i = tid; i < SMM; i += T) sh.cnt[i] = g_cnt[i];
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
        sh.best[0] = sh.best[1] = sh.best[2] = kNoKey;
    }
    if (tid < 2 * kMaxCluster) sh.rec[tid / kMaxCluster][tid % kMaxCluster].key = kNoKey;
    if (FAST) {
        // index offset of neighbour e of a site with basis index b when no periodic wrap occurs
        const int Ly = P.L[1], Lz = P.L[2];
        for (int i = tid; i < P.A * Z; i += T) {
            const int8_t* st = P.tab->stencil + i * 4;
            const int b = i / Z;
            s_ds[i] = (((int)st[1] * Ly + (int)st[2]) * Lz + (int)st[3]) * P.A + ((int)st[0] - b);
        }
        // interior sites: every cell coordinate in [1, L-2], so no neighbour (cell shifts are -1, 0, +1) wraps
        const int n_words = (N + 31) >> 5;
        for (int wd = tid >> 5; wd < n_words; wd += T >> 5) {
            const int site = wd * 32 + (tid & 31);
            const int cell = site / P.A;
            const int cz = cell % Lz, cy = (cell / Lz) % Ly, cx = cell / (Lz * Ly);
            const bool in = site < N && cx >= 1 && cx <= P.L[0] - 2 && cy >= 1 && cy <= Ly - 2 && cz >= 1 && cz <= Lz - 2;
            const uint32_t word = __ballot_sync(0xFFFFFFFFu, in);
            if ((tid & 31) == 0) s_bm[wd] = word;
        }
    }
    __syncthreads();
    if (tid == 0) {
        double J = 0.0;
        for (int s = 0; s < S; ++s)
            J = __dadd_rn(J, __dmul_rn(Kc.w[s], shell_sum<M, false>(sh.cnt + s * MM, Kc.g + s * MM, Kc.t + s * MM, Pack<M>::bias(), 0, 0)));
        sh.J = J;
    }
    if (R > 1) cg::this_cluster().sync(); else __syncthreads();   // peers' shared memory is initialised before any post

    const OccView<OCC> occ{OCC == OCC_GLOBAL ? g_occ : s_occ};
    const int32_t* __restrict__ nbr = P.nbr_site;
    const int zq0 = P.zoff[1] >> 1, zq1 = P.zoff[2] >> 1, zq2 = P.zoff[3] >> 1;   // shell boundaries in int2 units (z even)

    // this thread's candidates in a window: c = gtid + j*GT, j = 0, 1, ...; kept as (window step, k)
    const uint32_t GT = (uint32_t)T * (uint32_t)R;
    const uint32_t gtid = (uint32_t)tid * (uint32_t)R + rank;
    const uint32_t ts_first = gtid / (uint32_t)K, k_first = gtid - ts_first * (uint32_t)K;
    const uint32_t ts_inc = GT / (uint32_t)K, k_inc = GT - ts_inc * (uint32_t)K;
    // window cap: at most kMaxRounds candidates per thread (W = 1 is always allowed: K <= 1024 <= 32 * 32)
    uint32_t w_cap = (uint32_t)(((uint64_t)kMaxRounds * GT) / (uint32_t)K);
    if (w_cap < 1u) w_cap = 1u;
    if (w_cap > (uint32_t)A.w_max) w_cap = (uint32_t)A.w_max;
    if (w_cap > (1u << 20)) w_cap = 1u << 20;

    unsigned long long t0 = A.step0;
    const unsigned long long t_end = A.step0 + A.n_steps;
    uint32_t W = 1;
    unsigned long long my_null = 0;
    uint32_t it = 0;

    while (t0 < t_end) {
        const uint32_t Wc = (uint32_t)min((unsigned long long)W, t_end - t0);
        const int buf = (int)(it % 3u);
        volatile uint32_t* best_slot = &sh.best[buf];
        const double J_cur = sh.J;
        uint32_t win_key = kNoKey, win_a = 0, win_b = 0, win_pq = 0;
        PW win_d0 = 0, win_d1 = 0, win_d2 = 0;
        double win_J = 0.0;
        uint64_t nullmask = 0;

        uint32_t ts = ts_first, k = k_first;
        for (int j = 0; ts < Wc; ++j) {
            const uint32_t hint = *best_slot;
            if ((hint >> 10) < ts) break;                       // a move at an earlier step exists: this step is void
            const uint32_t key = (ts << 10) | k;
            // ---- D9.1 proposal
            const unsigned long long step = t0 + ts;
            const uint4 r = philox4x32_10((uint32_t)step, (uint32_t)(step >> 32), k, chain, key0, key1);
            uint32_t a = __umulhi(r.x, (uint32_t)N), b = __umulhi(r.y, (uint32_t)N - 1u);
            b += (b >= a);
            uint32_t p = occ.get(a), q = occ.get(b);
            if (p == q) {
                a = __umulhi(r.z, (uint32_t)N); b = __umulhi(r.w, (uint32_t)N - 1u);
                b += (b >= a);
                p = occ.get(a); q = occ.get(b);
            }
            if (p == q) {
                nullmask |= 1ull << j;
            } else if (key < hint) {                             // same step, higher k than a known move: only nullness counts
                // ---- D9.2 integer delta: per shell  sum_{nbrs of b} e_r - sum_{nbrs of a} e_r  (a, b excluded)
                // No per-entry exclusion: with m = #(entries of row a equal to b) and m_self = #(entries of a row equal
                // to its own site) -- the table is symmetric with multiplicity and every site is equivalent -- the
                // excluded sum is  d_all + (m - m_self) (e_q - e_p).
                PW d0 = 0, d1 = 0, d2 = 0;
                const int2* __restrict__ ra = reinterpret_cast<const int2*>(nbr + (size_t)a * Z);
                const int2* __restrict__ rb = reinterpret_cast<const int2*>(nbr + (size_t)b * Z);
                const bool ia = FAST && ((s_bm[a >> 5] >> (a & 31u)) & 1u), ib = FAST && ((s_bm[b >> 5] >> (b & 31u)) & 1u);
                const int2* da = reinterpret_cast<const int2*>(s_ds + (a & (uint32_t)(P.A - 1)) * Z);
                const int2* db = reinterpret_cast<const int2*>(s_ds + (b & (uint32_t)(P.A - 1)) * Z);
                const PW eqp = Pack<M>::one(q) - Pack<M>::one(p);
                auto shell = [&](int e0, int e1, int m_self) {
                    PW d = 0;
                    int m = -m_self;
#pragma unroll 3
                    for (int e = e0; e < e1; ++e) {
                        int2 va, vb;
                        if (ia) { const int2 o = da[e]; va = make_int2((int)a + o.x, (int)a + o.y); } else va = __ldg(ra + e);
                        if (ib) { const int2 o = db[e]; vb = make_int2((int)b + o.x, (int)b + o.y); } else vb = __ldg(rb + e);
                        d -= Pack<M>::one(occ.get((uint32_t)va.x));
                        d -= Pack<M>::one(occ.get((uint32_t)va.y));
                        d += Pack<M>::one(occ.get((uint32_t)vb.x));
                        d += Pack<M>::one(occ.get((uint32_t)vb.y));
                        m += ((uint32_t)va.x == b) + ((uint32_t)va.y == b);
                    }
                    return d + (PW)m * eqp + Pack<M>::bias();
                };
                // ---- D6 objective from counts + delta, shell by shell.  With w_s >= 0 every partial sum is an exact
                // lower bound of J_k (each term is >= 0 and rounding is monotonic), so once it reaches J_cur the candidate
                // cannot improve and the remaining shells are skipped when no lane of the warp still needs them.
                const bool prune = A.prune != 0;
                d0 = shell(0, zq0, P.m_self[0]);
                double Jk = __dmul_rn(Kc.w[0], shell_sum<M, SYM>(sh.cnt, Kc.g, Kc.t, d0, (int)p, (int)q));
                Jk = __dadd_rn(0.0, Jk);
                if (S > 1 && (!prune || __any_sync(__activemask(), Jk < J_cur))) {
                    d1 = shell(zq0, zq1, P.m_self[1]);
                    Jk = __dadd_rn(Jk, __dmul_rn(Kc.w[1], shell_sum<M, SYM>(sh.cnt + MM, Kc.g + MM, Kc.t + MM, d1, (int)p, (int)q)));
                    if (S > 2 && (!prune || __any_sync(__activemask(), Jk < J_cur))) {
                        d2 = shell(zq1, zq2, P.m_self[2]);
                        Jk = __dadd_rn(Jk, __dmul_rn(Kc.w[2], shell_sum<M, SYM>(sh.cnt + 2 * MM, Kc.g + 2 * MM, Kc.t + 2 * MM, d2, (int)p, (int)q)));
                    } else if (S > 2) {
                        Jk = J_cur;                       // pruned: not improving
                    }
                } else if (S > 1) {
                    Jk = J_cur;
                }
                if (Jk < J_cur && win_key == kNoKey) {
                    win_key = key; win_a = a; win_b = b; win_pq = p | (q << 8);
                    win_d0 = d0; win_d1 = d1; win_d2 = d2; win_J = Jk;
                    atomicMin(&sh.best[buf], key);
                }
            }
            k += k_inc; ts += ts_inc;
            if (k >= (uint32_t)K) { k -= (uint32_t)K; ++ts; }
        }
        __syncthreads();                                        // B1: window evaluated, local minimum posted
        uint32_t key_best = sh.best[buf];
        if (tid == 0) sh.best[(buf + 2) % 3] = kNoKey;          // next user of that slot is two barriers away

        const int warp = tid >> 5, lane = tid & 31;
        const MoveRec* mv = nullptr;                            // the move to apply (in this block's shared memory)
        if (R > 1) {
            // post this block's best record into every replica's rec[parity][rank], then pick the global minimum
            const int par = (int)(it & 1u);
            const uint32_t owner_lane_mask = __ballot_sync(0xFFFFFFFFu, win_key == key_best && key_best != kNoKey);
            const bool poster = key_best != kNoKey ? owner_lane_mask != 0u : warp == 0;
            if (poster) {
                const int src = key_best != kNoKey ? __ffs((int)owner_lane_mask) - 1 : 0;
                MoveRec m;
                m.key = key_best;
                m.a = __shfl_sync(0xFFFFFFFFu, win_a, src); m.b = __shfl_sync(0xFFFFFFFFu, win_b, src);
                m.pq = __shfl_sync(0xFFFFFFFFu, win_pq, src); m.J = __shfl_sync(0xFFFFFFFFu, win_J, src);
                m.d[0] = __shfl_sync(0xFFFFFFFFu, (uint64_t)win_d0, src); m.d[1] = __shfl_sync(0xFFFFFFFFu, (uint64_t)win_d1, src);
                m.d[2] = __shfl_sync(0xFFFFFFFFu, (uint64_t)win_d2, src);
                if (lane < R) {
                    MoveRec* dst = cg::this_cluster().map_shared_rank(&sh.rec[par][rank], lane);
                    *dst = m;
                }
            }
            cg::this_cluster().sync();                          // release/acquire: all records visible in every replica
            uint32_t kb = kNoKey; int src_rank = 0;
            for (int r2 = 0; r2 < R; ++r2) {
                const uint32_t kk = sh.rec[par][r2].key;
                if (kk < kb) { kb = kk; src_rank = r2; }
            }
            key_best = kb;
            mv = &sh.rec[par][src_rank];
        } else if (key_best != kNoKey) {
            // single block: the owner's warp copies the record to shared memory for the cooperative apply
            const uint32_t owner_lane_mask = __ballot_sync(0xFFFFFFFFu, win_key == key_best);
            if (owner_lane_mask != 0u && lane == __ffs((int)owner_lane_mask) - 1) {
                MoveRec& m = sh.rec[0][0];
                m.key = key_best; m.a = win_a; m.b = win_b; m.pq = win_pq; m.J = win_J;
                m.d[0] = win_d0; m.d[1] = win_d1; m.d[2] = win_d2;
            }
            __syncthreads();
            mv = &sh.rec[0][0];
        }

        // ---- commit: null counts of the committed steps, then the move (D9.4)
        const uint32_t steps_done = key_best != kNoKey ? (key_best >> 10) + 1u : Wc;
        if (nullmask) {
            const uint32_t lim = steps_done * (uint32_t)K;       // candidates c < lim are committed
            const uint32_t n_comm = gtid < lim ? (lim - 1u - gtid) / GT + 1u : 0u;
            my_null += __popcll(n_comm >= 64u ? nullmask : (nullmask & ((1ull << n_comm) - 1ull)));
        }
        if (key_best != kNoKey) {
            const int p = (int)(mv->pq & 0xFFu), q = (int)(mv->pq >> 8);
            for (int idx = tid; idx < SMM; idx += T) {
                const int s = idx / MM, rem = idx - s * MM, i = rem / M, jj = rem - i * M;
                const PW d = (PW)mv->d[s];
                const int ci = (i == p) - (i == q), cj = (jj == p) - (jj == q);
                sh.cnt[idx] += ci * Pack<M>::field(d, jj) + cj * Pack<M>::field(d, i);
            }
            if (tid == T - 1) {                                 // one thread (not among the count updaters when T > SMM)
                const uint32_t a = mv->a, b = mv->b, kk = key_best & 1023u;
                const unsigned long long step = t0 + (key_best >> 10);
                if (OCC != OCC_GLOBAL || rank == 0) { occ.set(a, (uint32_t)q); occ.set(b, (uint32_t)p); }
                sh.J = mv->J;
                sh.n_accept += 1;
                sh.last_accept = step;
                unsigned long long h = sh.hash;
                h = (h ^ (uint32_t)step) * 0x100000001b3ULL;
                h = (h ^ (uint32_t)(step >> 32)) * 0x100000001b3ULL;
                h = (h ^ kk) * 0x100000001b3ULL;
                h = (h ^ a) * 0x100000001b3ULL;
                h = (h ^ b) * 0x100000001b3ULL;
                sh.hash = h;
                const unsigned long long nl = sh.n_logged;
                if (rank == 0 && A.log_all != nullptr && (long long)nl < A.log_cap) {
                    unsigned long long* rec = A.log_all + (chain_local * (size_t)A.log_cap + nl) * 3;
                    rec[0] = step;
                    rec[1] = (unsigned long long)kk | ((unsigned long long)a << 32);
                    rec[2] = (unsigned long long)b;
                }
                sh.n_logged = nl + 1;
            }
            // the move must be visible before the next window's reads; with a global occupancy shared by a cluster
            // the writer is rank 0, so the whole cluster waits
            if (OCC == OCC_GLOBAL && R > 1) cg::this_cluster().sync(); else __syncthreads();
            W = min(steps_done, w_cap);                         // the observed gap
        } else {
            W = min(W * 2u, w_cap);
        }
        t0 += steps_done;
        ++it;
    }

    // ---- epilogue: write back (rank 0 owns the global copy; null counts are summed over the blocks)
    if (my_null) atomicAdd(&sh.n_null, my_null);
    __syncthreads();
    if (rank == 0) {
        if (OCC == OCC_SMEM_U8) {
            for (int i = tid; i < N; i += T) g_occ[i] = s_occ[i];
        } else if (OCC == OCC_SMEM_NIB) {
            for (int i = tid; i < N; i += T) g_occ[i] = (uint8_t)occ.get(i);
        }
        for (int i = tid; i < SMM; i += T) g_cnt[i] = sh.cnt[i];
        if (tid == 0) {
            g_stats[0] = sh.n_accept;
            g_stats[2] = sh.hash;
            g_stats[3] = sh.last_accept;
            g_stats[4] = (unsigned long long)__double_as_longlong(sh.J);
        }
    }
    if (tid == 0 && sh.n_null) atomicAdd(&g_stats[1], sh.n_null);
}

// query != nullptr: no launch, *query = how many clusters of A.R blocks of this shape can be resident at once.
template <int M, int OCC, bool SYM>
cudaError_t launch_one(const KParams& P, const DevTables& host_tab, const McArgs& A, int64_t C, int threads,
                       size_t smem, cudaStream_t st, int* query)
{
    McConst<M> Kc;
    for (int s = 0; s < 3; ++s)
        for (int i = 0; i < M * M; ++i) {
            Kc.g[s * M * M + i] = s < P.S ? host_tab.g[s * M * M + i] : 0.0;
            Kc.t[s * M * M + i] = s < P.S ? host_tab.t[s * M * M + i] : 0.0;
        }
    for (int s = 0; s < 4; ++s) Kc.w[s] = host_tab.w[s];
    auto kern = mc_window_kernel<M, OCC, SYM>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(C * A.R));
    cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)A.R;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (query) return cudaOccupancyMaxActiveClusters(query, kern, &cfg);
    return cudaLaunchKernelEx(&cfg, kern, P, Kc, A);
}

template <int M, bool SYM>
cudaError_t launch_occ(int occ_mode, const KParams& P, const DevTables& host_tab, const McArgs& A, int64_t C,
                       int threads, size_t smem, cudaStream_t st, int* query)
{
    switch (occ_mode) {
        case OCC_SMEM_U8: return launch_one<M, OCC_SMEM_U8, SYM>(P, host_tab, A, C, threads, smem, st, query);
        case OCC_SMEM_NIB: return launch_one<M, OCC_SMEM_NIB, SYM>(P, host_tab, A, C, threads, smem, st, query);
        default: return launch_one<M, OCC_GLOBAL, SYM>(P, host_tab, A, C, threads, smem, st, query);
    }
}

template <int M>
cudaError_t launch_sym(bool sym, int occ_mode, const KParams& P, const DevTables& host_tab, const McArgs& A, int64_t C,
                       int threads, size_t smem, cudaStream_t st, int* query)
{
    return sym ? launch_occ<M, true>(occ_mode, P, host_tab, A, C, threads, smem, st, query)
               : launch_occ<M, false>(occ_mode, P, host_tab, A, C, threads, smem, st, query);
}

}  // namespace

size_t mc_shared_bytes(int occ_mode, int N, int AZ, bool fast_nbr)
{
    size_t s = sizeof(ChainShared) + sizeof(int) * (size_t)((AZ + 3) & ~3);
    if (fast_nbr && occ_mode != OCC_GLOBAL) s += sizeof(uint32_t) * (size_t)(((N + 127) >> 7) << 2);
    if (occ_mode == OCC_SMEM_U8) s += (size_t)N;
    else if (occ_mode == OCC_SMEM_NIB) s += (size_t)(N + 1) / 2;
    return (s + 15) & ~(size_t)15;
}

cudaError_t launch_mc(const KParams& P, const DevTables& host_tab, int occ_mode, int threads, int cluster, int w_max,
                      bool fast_nbr, uint8_t* occ, int32_t* counts, int64_t C, uint64_t n_steps, int K, uint64_t seed, uint64_t chain0,
                      uint64_t step0, void* stats, void* log, int64_t log_cap, cudaStream_t st, int64_t* n_launches,
                      int* query_max_clusters)
{
    const size_t smem = mc_shared_bytes(occ_mode, P.N, P.A * P.Z, fast_nbr);
    McArgs A;
    A.occ_all = occ; A.counts_all = counts;
    A.n_steps = n_steps; A.seed = seed; A.chain0 = chain0; A.step0 = step0;
    A.stats_all = reinterpret_cast<unsigned long long*>(stats);
    A.log_all = reinterpret_cast<unsigned long long*>(log);
    A.log_cap = log_cap; A.K = K; A.R = cluster; A.w_max = w_max; A.fast_nbr = fast_nbr ? 1 : 0;
    // exact pruning needs every shell term to be >= 0; the symmetric evaluation needs t_ij == t_ji bit for bit
    bool sym = true;
    A.prune = 1;
    for (int s = 0; s < P.S; ++s) {
        if (!(host_tab.w[s] >= 0.0)) A.prune = 0;
        for (int i = 0; i < P.M; ++i)
            for (int j = 0; j < i; ++j) {
                const double x = host_tab.t[(s * P.M + i) * P.M + j], y = host_tab.t[(s * P.M + j) * P.M + i];
                if (memcmp(&x, &y, sizeof(double)) != 0) sym = false;
            }
    }
    cudaError_t e;
    switch (P.M) {
        case 1: e = launch_sym<1>(sym, occ_mode, P, host_tab, A, C, threads, smem, st, query_max_clusters); break;
        case 2: e = launch_sym<2>(sym, occ_mode, P, host_tab, A, C, threads, smem, st, query_max_clusters); break;
        case 3: e = launch_sym<3>(sym, occ_mode, P, host_tab, A, C, threads, smem, st, query_max_clusters); break;
        case 4: e = launch_sym<4>(sym, occ_mode, P, host_tab, A, C, threads, smem, st, query_max_clusters); break;
        case 5: e = launch_sym<5>(sym, occ_mode, P, host_tab, A, C, threads, smem, st, query_max_clusters); break;
        case 6: e = launch_sym<6>(sym, occ_mode, P, host_tab, A, C, threads, smem, st, query_max_clusters); break;
        case 7: e = launch_sym<7>(sym, occ_mode, P, host_tab, A, C, threads, smem, st, query_max_clusters); break;
        default: e = launch_sym<8>(sym, occ_mode, P, host_tab, A, C, threads, smem, st, query_max_clusters); break;
    }
    if (e == cudaSuccess && !query_max_clusters) ++*n_launches;
    return e;
}

}  // namespace hea
