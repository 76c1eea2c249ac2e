// hea_sro.cu -- full Warren-Cowley recount (hea_sro_full) and seeded initial placement (hea_init_random).
// DESIGN.md D4-D6, D8; Eq. 2, Eq. 3, P:207, P:275 (the recount is >99% of the
// time of the non-incremental search).
//
// Recount kernel.  HBM-bound by the neighbour table: 4*Z bytes per site per pass, plus one occupancy byte.
//   - the site-major table [Npad][Z] is streamed through shared memory with bulk asynchronous copies
//     (cp.async.bulk global -> shared, completion on an mbarrier): a TILE is 32 consecutive sites = one contiguous
//     128*Z-byte run of the table = one copy.  Every WARP owns a private ring of stages and its own mbarriers; lane 0
//     refills a stage as soon as the warp has consumed it, so there is no block-level synchronisation in the main loop
//     and the bytes in flight per SM (warps x stages x 128 Z) are set by shared memory, not by registers;
//   - lane = site of the tile: it reads its table row from shared memory as 8-byte words (row stride 4 Z bytes, Z even
//     but Z/2 odd or = 2 mod 4 for every supported lattice/shell set: conflict-free or 2-way), gathers the Z neighbour
//     species bytes (neighbours of consecutive sites are consecutive: one or two 32-byte sectors per warp gather,
//     L1/L2 hits) with all gathers of a site in flight at once (shell sizes are template constants);
//   - per site and shell the neighbour species are counted in a packed register histogram, then folded into per-thread
//     rows acc[s][own species] of 16-bit fields with multiply-adds by the 0/1 "row is mine" flags (no dynamic
//     register indexing);
//   - at the end: unpack, warp REDUX add, shared-memory bins, one global atomicAdd per bin per block.
// A block walks a contiguous range of tiles (its warps interleaved), so the occupancy lines it gathers from form a
// few sliding windows that stay in L1.  Integer adds commute, so the result is bit-exact whatever the order.
#include <algorithm>
#include <type_traits>

#include "hea_device.cuh"

namespace hea {

namespace {

constexpr int kSroMaxWarps = 16;
constexpr int kSroMaxThreads = kSroMaxWarps * 32;
constexpr int kSroMaxStages = 8;
constexpr int kFlushTiles = 2048;         // 16-bit fields: 2048 sites per lane * z <= 24 < 65536

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

// arm the barrier with the byte count, then start the bulk copy that completes on it
__device__ __forceinline__ void bulk_load(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "HEA_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra HEA_DONE_%=;\n"
        "bra HEA_WAIT_%=;\n"
        "HEA_DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}

// Packed per-site neighbour histogram of one shell (counts <= 24): M <= 4 -> 8-bit fields in 32 bits, M == 5 -> 6-bit
// fields in 32 bits, M >= 6 -> 8-bit fields in 64 bits.  spread16(w) = fields 2w and 2w+1 as two 16-bit fields.
template <int M>
struct Hist {
    static constexpr int FB = (M == 5) ? 6 : 8;
    using W = typename std::conditional<(M * FB <= 32), uint32_t, uint64_t>::type;
    __device__ __forceinline__ static W one(uint32_t species) { return (W)1 << (FB * species); }
    __device__ __forceinline__ static uint32_t spread16(W h, int w)
    {
        if (FB == 8) {
            const uint32_t half = (w < 2) ? (uint32_t)h : (uint32_t)((uint64_t)h >> 32);
            return __byte_perm(half, 0, (w & 1) ? 0x4342 : 0x4140);
        }
        const uint32_t x = (uint32_t)h >> (12 * w);
        return (x & 63u) | ((x << 10) & (63u << 16));
    }
};

// LAT 0 = fcc (z = 12, 6, 24), 1 = bcc (z = 8, 6, 12): D2.
template <int LAT, int S>
struct Shells {
    static constexpr int z0 = LAT == 0 ? 12 : 8, z1 = S > 1 ? 6 : 0, z2 = S > 2 ? (LAT == 0 ? 24 : 12) : 0;
    static constexpr int Z = z0 + z1 + z2;
};

template <int M, int LAT, int S>
__global__ void __launch_bounds__(kSroMaxThreads)
sro_count_kernel(const KParams P, const uint8_t* __restrict__ occ_all, int32_t* __restrict__ counts_all,
                 int tiles_per_block, int n_stages)
{
    using SH = Shells<LAT, S>;
    using H = Hist<M>;
    using HW = typename H::W;
    constexpr int Z = SH::Z, ZH = Z / 2;
    constexpr int W16 = (M + 1) / 2;      // 32-bit words per accumulator row, two 16-bit fields (species 2w, 2w+1) each
    constexpr uint32_t kStageBytes = 128u * Z;

    extern __shared__ __align__(128) uint8_t s_stage[];              // [warp][stage][32 sites][Z] int32
    __shared__ uint64_t s_bar[kSroMaxWarps * kSroMaxStages];
    __shared__ int s_bins[kSMM];
    constexpr int SMM = S * M * M;
    for (int i = threadIdx.x; i < SMM; i += blockDim.x) s_bins[i] = 0;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int kSroWarps = (int)(blockDim.x >> 5);
    const uint8_t* __restrict__ occ = occ_all + (size_t)blockIdx.y * P.N;
    const int n_tiles = P.Npad >> 5;
    const int t_begin = blockIdx.x * tiles_per_block;
    const int t_end = min(n_tiles, t_begin + tiles_per_block);
    uint8_t* my_stage = s_stage + (size_t)warp * n_stages * kStageBytes;
    uint64_t* my_bar = s_bar + warp * kSroMaxStages;
    const uint8_t* tab = reinterpret_cast<const uint8_t*>(P.nbr_site);

    // this warp's tiles: t_begin + warp + i * kSroWarps
    const int first = t_begin + warp;
    const int n_mine = first < t_end ? (t_end - first + kSroWarps - 1) / kSroWarps : 0;
    if (lane == 0) {
        for (int st = 0; st < n_stages; ++st) mbar_init(my_bar + st, 1);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        for (int st = 0; st < n_stages && st < n_mine; ++st)
            bulk_load(my_stage + (size_t)st * kStageBytes, tab + (size_t)(first + st * kSroWarps) * kStageBytes,
                      kStageBytes, my_bar + st);
    }
    __syncthreads();                                                  // s_bins zeroed, barriers initialised

    uint32_t acc[S][M][W16];
#pragma unroll
    for (int s = 0; s < S; ++s)
#pragma unroll
        for (int i = 0; i < M; ++i)
#pragma unroll
            for (int w = 0; w < W16; ++w) acc[s][i][w] = 0;

    auto flush = [&]() {
#pragma unroll
        for (int s = 0; s < S; ++s)
#pragma unroll
            for (int i = 0; i < M; ++i)
#pragma unroll
                for (int j = 0; j < M; ++j) {
                    const int v = (acc[s][i][j >> 1] >> ((j & 1) * 16)) & 0xFFFF;
                    const int tot = __reduce_add_sync(0xFFFFFFFFu, v);
                    if (lane == 0 && tot) atomicAdd(&s_bins[(s * M + i) * M + j], tot);
                }
#pragma unroll
        for (int s = 0; s < S; ++s)
#pragma unroll
            for (int i = 0; i < M; ++i)
#pragma unroll
                for (int w = 0; w < W16; ++w) acc[s][i][w] = 0;
    };

    int since_flush = 0;
    int st = 0;
    uint32_t parity = 0;
    for (int i = 0; i < n_mine; ++i) {
        const int tile = first + i * kSroWarps;
        const int site = (tile << 5) + lane;
        const uint32_t own = site < P.N ? (uint32_t)__ldg(occ + site) : 0xFFu;   // 0xFF matches no row
        uint32_t mine[M];
#pragma unroll
        for (int r = 0; r < M; ++r) mine[r] = own == (uint32_t)r;
        mbar_wait(my_bar + st, parity);
        const int2* __restrict__ row = reinterpret_cast<const int2*>(my_stage + (size_t)st * kStageBytes) + lane * ZH;
        int2 nb[ZH];
#pragma unroll
        for (int e = 0; e < ZH; ++e) nb[e] = row[e];
        uint32_t sp[Z];
#pragma unroll
        for (int e = 0; e < ZH; ++e) {
            sp[2 * e] = __ldg(occ + (uint32_t)nb[e].x);
            sp[2 * e + 1] = __ldg(occ + (uint32_t)nb[e].y);
        }
        // the stage is consumed (its words are in registers): refill it with the tile n_stages ahead
        __syncwarp();
        if (lane == 0 && i + n_stages < n_mine)
            bulk_load(my_stage + (size_t)st * kStageBytes, tab + (size_t)(tile + n_stages * kSroWarps) * kStageBytes,
                      kStageBytes, my_bar + st);
        if (++st == n_stages) { st = 0; parity ^= 1u; }
#pragma unroll
        for (int s = 0; s < S; ++s) {
            constexpr int zo[4] = {0, SH::z0, SH::z0 + SH::z1, SH::Z};
            HW h = 0;
#pragma unroll
            for (int e = zo[s]; e < zo[s + 1]; ++e) h += H::one(sp[e]);
#pragma unroll
            for (int w = 0; w < W16; ++w) {
                const uint32_t e16 = H::spread16(h, w);
#pragma unroll
                for (int r = 0; r < M; ++r) acc[s][r][w] += e16 * mine[r];
            }
        }
        if (++since_flush >= kFlushTiles) { flush(); since_flush = 0; }          // warp-uniform
    }
    flush();
    __syncthreads();
    int32_t* counts = counts_all + (size_t)blockIdx.y * SMM;
    for (int i = threadIdx.x; i < SMM; i += blockDim.x) {
        const int v = s_bins[i];
        if (v) atomicAdd(&counts[i], v);
    }
}

// alpha (Eq. 2) and J (Eq. 3) from the integer counts, in the D6 order.  One thread per configuration.
__global__ void sro_epilogue_kernel(const KParams P, const int32_t* __restrict__ counts_all, int64_t B,
                                    double* __restrict__ alpha_all, double* __restrict__ obj)
{
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const int M = P.M, SMM = P.S * M * M;
    const int32_t* counts = counts_all + b * SMM;
    const DevTables* T = P.tab;
    double J = 0.0;
    for (int s = 0; s < P.S; ++s) {
        double sh = 0.0;
        for (int i = 0; i < M; ++i) {
            double row = 0.0;
            for (int j = 0; j < M; ++j) {
                const int idx = (s * M + i) * M + j;
                const int n = counts[idx];
                if (alpha_all) alpha_all[b * SMM + idx] = __dsub_rn(1.0, __dmul_rn((double)n, T->g[idx]));
                row = __dadd_rn(row, sq_dev(n, T->g[idx], T->t[idx]));
            }
            sh = __dadd_rn(sh, row);
        }
        J = __dadd_rn(J, __dmul_rn(T->w[s], sh));
    }
    if (obj) obj[b] = J;
}

// ---------------------------------------------------------------- D8: seeded Fisher-Yates
// One block per chain.  The Philox draws are independent and are produced by all threads in chunks; the swaps are a
// serial dependency chain, applied by warp 0 in groups of 32 that touch disjoint sites (one swap per lane; a group with
// a collision is applied in order by lane 0) -- in shared memory when the configuration fits, else in global memory.
constexpr int kInitThreads = 256;
constexpr int kInitChunk = 2048;

template <bool IN_SMEM>
__global__ void __launch_bounds__(kInitThreads)
init_random_kernel(const KParams P, uint8_t* __restrict__ occ_all, uint64_t seed, uint64_t chain0,
                   const int64_t* __restrict__ n_per_species)
{
    extern __shared__ __align__(16) uint8_t s_raw[];
    uint32_t* s_j = reinterpret_cast<uint32_t*>(s_raw);             // [kInitChunk]
    uint8_t* s_occ = s_raw + kInitChunk * sizeof(uint32_t);          // [N] when IN_SMEM
    uint8_t* g_occ = occ_all + (size_t)blockIdx.x * P.N;
    uint8_t* o = IN_SMEM ? s_occ : g_occ;
    const uint32_t chain = (uint32_t)(chain0 + blockIdx.x);
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);

    // species blocks in ascending order
    int64_t bound[9];
    bound[0] = 0;
    for (int i = 0; i < P.M; ++i) bound[i + 1] = bound[i] + n_per_species[i];
    for (int n = threadIdx.x; n < P.N; n += blockDim.x) {
        int sp = 0;
        while (n >= bound[sp + 1]) ++sp;
        o[n] = (uint8_t)sp;
    }
    __syncthreads();

    for (int hi = P.N - 1; hi >= 1; hi -= kInitChunk) {
        const int lo = max(1, hi - kInitChunk + 1);                  // this chunk handles n = hi .. lo
        for (int i = threadIdx.x; i <= hi - lo; i += blockDim.x) {
            const uint32_t n = (uint32_t)(hi - i);
            const uint4 r = philox4x32_10(n, 0u, 0xFFFFFFFFu, chain, k0, k1);
            s_j[i] = __umulhi(r.x, n + 1u);
        }
        __syncthreads();
        // The swaps are a serial chain, but 32 consecutive ones commute when they touch disjoint sites: all j distinct and
        // no j inside the group's own range of n (other than j = n, a no-op).  Warp 0 applies such a group with one swap
        // per lane (32 random accesses in flight instead of one); a group with a collision is applied in order by lane 0.
        // Collisions are likely only while n is small (~1500 / n per group).  Same result as the serial order, bit for bit.
        if (threadIdx.x < 32) {
            const int lane = threadIdx.x;
            const int cnt = hi - lo + 1;
            for (int i0 = 0; i0 < cnt; i0 += 32) {
                const int i = i0 + lane;
                const bool have = i < cnt;
                const int n = hi - i;
                const uint32_t j = have ? s_j[i] : 0xFFFFFFFFu - (uint32_t)lane;     // idle lanes: distinct dummies
                const int n_lo = hi - min(i0 + 31, cnt - 1);                             // the group covers n_lo .. hi - i0
                const uint32_t same_j = __match_any_sync(0xFFFFFFFFu, j);              // every lane takes part
                const bool clash = have && (same_j != (1u << lane) || (j >= (uint32_t)n_lo && j != (uint32_t)n));
                if (!__any_sync(0xFFFFFFFFu, clash)) {
                    if (have) {
                        const uint8_t a = o[n], b = o[j];
                        o[n] = b; o[j] = a;
                    }
                } else if (lane == 0) {
                    for (int k = i0; k < min(i0 + 32, cnt); ++k) {
                        const int nn = hi - k;
                        const uint32_t jj = s_j[k];
                        const uint8_t a = o[nn], b = o[jj];
                        o[nn] = b; o[jj] = a;
                    }
                }
                __syncwarp();
            }
        }
        __syncthreads();
    }
    if (IN_SMEM)
        for (int n = threadIdx.x; n < P.N; n += blockDim.x) g_occ[n] = s_occ[n];
}

__global__ void stats_reset_kernel(uint64_t* stats_words, int64_t C)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= C) return;
    uint64_t* st = stats_words + c * 5;
    st[0] = 0; st[1] = 0; st[2] = 0xcbf29ce484222325ULL; st[3] = 0xffffffffffffffffULL; st[4] = 0;   // J = +0.0
}

}  // namespace

// ---------------------------------------------------------------- launchers (called from hea_api.cu)
namespace {

template <int M, int LAT, int S>
cudaError_t launch_sro_one(const KParams& P, const uint8_t* occ, int32_t* counts, dim3 grid, int tiles_per_block,
                           int n_stages, int n_warps, cudaStream_t st)
{
    auto kern = sro_count_kernel<M, LAT, S>;
    const size_t smem = (size_t)n_stages * n_warps * 128u * Shells<LAT, S>::Z;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, n_warps * 32, smem, st>>>(P, occ, counts, tiles_per_block, n_stages);
    return cudaGetLastError();
}

template <int M>
cudaError_t launch_sro_m(const KParams& P, int lat, const uint8_t* occ, int32_t* counts, dim3 grid, int tiles_per_block,
                         int n_stages, int n_warps, cudaStream_t st)
{
    switch (lat * 3 + P.S) {
        case 1: return launch_sro_one<M, 0, 1>(P, occ, counts, grid, tiles_per_block, n_stages, n_warps, st);
        case 2: return launch_sro_one<M, 0, 2>(P, occ, counts, grid, tiles_per_block, n_stages, n_warps, st);
        case 3: return launch_sro_one<M, 0, 3>(P, occ, counts, grid, tiles_per_block, n_stages, n_warps, st);
        case 4: return launch_sro_one<M, 1, 1>(P, occ, counts, grid, tiles_per_block, n_stages, n_warps, st);
        case 5: return launch_sro_one<M, 1, 2>(P, occ, counts, grid, tiles_per_block, n_stages, n_warps, st);
        default: return launch_sro_one<M, 1, 3>(P, occ, counts, grid, tiles_per_block, n_stages, n_warps, st);
    }
}

}  // namespace

// lat: 0 fcc, 1 bcc (the shell sizes are template constants of the kernel).  smem_budget: opt-in shared memory per block.
cudaError_t launch_sro_count(const KParams& P, int lat, const uint8_t* occ, int64_t B, int32_t* counts, int n_sms,
                             size_t smem_budget, int opt_stages, int opt_blocks_per_sm, int opt_warps, cudaStream_t st, int64_t* n_launches)
{
    const int SMM = P.S * P.M * P.M;
    cudaError_t e = cudaMemsetAsync(counts, 0, sizeof(int32_t) * (size_t)SMM * (size_t)B, st);
    if (e != cudaSuccess) return e;
    const int n_tiles = P.Npad >> 5;
    const int kSroWarps = opt_warps > 0 ? opt_warps : 16, n_warps = kSroWarps;
    const size_t stage_bytes = (size_t)kSroWarps * 128u * P.Z;      // one stage of every warp of a block
    // resident blocks per SM (default one block of 16 warps; measured within 2 % of 2 x 8 warps on B200), each with an
    // equal share of the SM's shared memory for its stage ring; at least one stage per warp must fit
    const size_t per_sm = smem_budget + 1024;                       // opt-in per-block limit + its 1 KB reservation
    int bps = opt_blocks_per_sm > 0 ? opt_blocks_per_sm : 1;
    while (bps > 1 && per_sm / bps < stage_bytes + 5120) --bps;
    const size_t usable = per_sm / bps > 5120 ? per_sm / bps - 5120 : 0;   // static (barriers, bins) + reservation
    int max_stages = (int)std::min<size_t>(kSroMaxStages, usable / stage_bytes);
    if (max_stages < 1) return cudaErrorInvalidConfiguration;
    if (opt_stages > 0 && opt_stages < max_stages) max_stages = opt_stages;
    // blocks per configuration: bps blocks per SM over the whole batch, each walking a contiguous range of tiles
    int64_t bx = std::max<int64_t>(1, (int64_t)n_sms * bps / std::max<int64_t>(1, B));
    bx = std::min<int64_t>(bx, (n_tiles + kSroWarps - 1) / kSroWarps);
    const int tiles_per_block = (int)((n_tiles + bx - 1) / bx);
    bx = (n_tiles + tiles_per_block - 1) / tiles_per_block;
    const int n_stages = std::max(1, std::min(max_stages, (tiles_per_block + kSroWarps - 1) / kSroWarps));
    for (int64_t b0 = 0; b0 < B; b0 += 65535) {
        const int by = (int)((B - b0) < 65535 ? (B - b0) : 65535);
        dim3 grid((unsigned)bx, by);
        const uint8_t* o = occ + (size_t)b0 * P.N;
        int32_t* c = counts + (size_t)b0 * SMM;
        switch (P.M) {
            case 1: e = launch_sro_m<1>(P, lat, o, c, grid, tiles_per_block, n_stages, n_warps, st); break;
            case 2: e = launch_sro_m<2>(P, lat, o, c, grid, tiles_per_block, n_stages, n_warps, st); break;
            case 3: e = launch_sro_m<3>(P, lat, o, c, grid, tiles_per_block, n_stages, n_warps, st); break;
            case 4: e = launch_sro_m<4>(P, lat, o, c, grid, tiles_per_block, n_stages, n_warps, st); break;
            case 5: e = launch_sro_m<5>(P, lat, o, c, grid, tiles_per_block, n_stages, n_warps, st); break;
            case 6: e = launch_sro_m<6>(P, lat, o, c, grid, tiles_per_block, n_stages, n_warps, st); break;
            case 7: e = launch_sro_m<7>(P, lat, o, c, grid, tiles_per_block, n_stages, n_warps, st); break;
            default: e = launch_sro_m<8>(P, lat, o, c, grid, tiles_per_block, n_stages, n_warps, st); break;
        }
        if (e != cudaSuccess) return e;
        ++*n_launches;
    }
    return cudaSuccess;
}

cudaError_t launch_sro_epilogue(const KParams& P, const int32_t* counts, int64_t B, double* alpha, double* obj,
                                cudaStream_t st, int64_t* n_launches)
{
    if (!alpha && !obj) return cudaSuccess;
    const int threads = 64;
    sro_epilogue_kernel<<<(unsigned)((B + threads - 1) / threads), threads, 0, st>>>(P, counts, B, alpha, obj);
    ++*n_launches;
    return cudaGetLastError();
}

cudaError_t launch_init_random(const KParams& P, uint8_t* occ, int64_t C, uint64_t seed, uint64_t chain0,
                               const int64_t* n_per_species_dev, size_t smem_budget, cudaStream_t st, int64_t* n_launches)
{
    const size_t base = kInitChunk * sizeof(uint32_t);
    const bool in_smem = (size_t)P.N + base <= smem_budget;      // the device's opt-in shared memory per block
    cudaError_t e = cudaSuccess;
    if (in_smem) {
        e = cudaFuncSetAttribute(init_random_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(base + (size_t)P.N));
        if (e != cudaSuccess) return e;
    }
    const int64_t kMaxGrid = 0x7FFFFFFF;                          // gridDim.x limit: more chains go in several launches
    for (int64_t c0 = 0; c0 < C; c0 += kMaxGrid) {
        const unsigned grid = (unsigned)std::min<int64_t>(kMaxGrid, C - c0);
        uint8_t* o = occ + (size_t)c0 * (size_t)P.N;
        if (in_smem) init_random_kernel<true><<<grid, kInitThreads, base + (size_t)P.N, st>>>(P, o, seed, chain0 + (uint64_t)c0, n_per_species_dev);
        else init_random_kernel<false><<<grid, kInitThreads, base, st>>>(P, o, seed, chain0 + (uint64_t)c0, n_per_species_dev);
        ++*n_launches;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return e;
}

cudaError_t launch_stats_reset(void* stats, int64_t C, cudaStream_t st, int64_t* n_launches)
{
    stats_reset_kernel<<<(unsigned)((C + 255) / 256), 256, 0, st>>>(reinterpret_cast<uint64_t*>(stats), C);
    ++*n_launches;
    return cudaGetLastError();
}

}  // namespace hea
