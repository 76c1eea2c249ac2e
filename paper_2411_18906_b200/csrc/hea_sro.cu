// hea_sro.cu -- full Warren-Cowley recount (hea_sro_full) and seeded initial placement (hea_init_random).
// DESIGN.md D4-D6, D8; Eq. 2, Eq. 3, P:207, P:275 (the recount is >99% of the
// time of the non-incremental search).
//
// Recount kernel (direct variant).  HBM-bound by the slot-major neighbour table: 4*Z bytes per site per pass.
//   - one thread owns 4 consecutive sites; for every slot it reads the 4 neighbour indices with one 16-byte
//     coalesced load (a warp reads 512 contiguous bytes of the table per slot) and gathers the 4 neighbour species
//     bytes (lattice-local, L1/L2 hits);
//   - per site and shell the neighbour species are counted in a packed register histogram (8-bit fields), then
//     folded into per-thread rows acc[s][own species] of 16-bit fields with predicated adds (no dynamic indexing);
//   - at the end: unpack, warp REDUX add, shared-memory bins, one global atomicAdd per bin per block.
// Integer adds commute, so the result is bit-exact whatever the order.
#include "hea_device.cuh"

namespace hea {

namespace {

constexpr int kSroThreads = 256;
constexpr int kFlushSites = 2048;         // 16-bit fields: 2048 sites * z<=24 < 65536

template <int M>
__global__ void __launch_bounds__(kSroThreads)
sro_count_kernel(const KParams P, const uint8_t* __restrict__ occ_all, int32_t* __restrict__ counts_all)
{
    constexpr int W = (M + 1) / 2;        // 32-bit words per row, two 16-bit fields (species 2w, 2w+1) each
    __shared__ int s_bins[kSMM];
    const int SMM = P.S * M * M;
    for (int i = threadIdx.x; i < SMM; i += blockDim.x) s_bins[i] = 0;
    __syncthreads();

    const uint8_t* __restrict__ occ = occ_all + (size_t)blockIdx.y * P.N;
    const bool aligned4 = ((reinterpret_cast<uintptr_t>(occ) & 3) == 0);

    uint32_t acc[3][M][W];
#pragma unroll
    for (int s = 0; s < 3; ++s)
#pragma unroll
        for (int i = 0; i < M; ++i)
#pragma unroll
            for (int w = 0; w < W; ++w) acc[s][i][w] = 0;

    auto flush = [&]() {
#pragma unroll
        for (int s = 0; s < 3; ++s) {
            if (s < P.S) {
#pragma unroll
                for (int i = 0; i < M; ++i)
#pragma unroll
                    for (int j = 0; j < M; ++j) {
                        const int v = (acc[s][i][j >> 1] >> ((j & 1) * 16)) & 0xFFFF;
                        const int tot = __reduce_add_sync(0xFFFFFFFFu, v);
                        if ((threadIdx.x & 31) == 0 && tot) atomicAdd(&s_bins[(s * M + i) * M + j], tot);
                    }
            }
        }
#pragma unroll
        for (int s = 0; s < 3; ++s)
#pragma unroll
            for (int i = 0; i < M; ++i)
#pragma unroll
                for (int w = 0; w < W; ++w) acc[s][i][w] = 0;
    };

    const int n_quads = P.Npad >> 2;
    int since_flush = 0;
    const int lane = threadIdx.x & 31;
    // warp-uniform trip count (flush() uses full-warp REDUX): lanes past the end work on quad 0 with a species
    // id that matches no row, so they add nothing.
    for (int quad = blockIdx.x * blockDim.x + threadIdx.x; quad - lane < n_quads; quad += gridDim.x * blockDim.x) {
        const bool active = quad < n_quads;
        const int site0 = active ? quad << 2 : 0;
        const int n_valid = active ? min(4, P.N - site0) : 0;
        uint32_t own[4];
        if (aligned4 && n_valid == 4) {
            const uint32_t o4 = *reinterpret_cast<const uint32_t*>(occ + site0);
            own[0] = o4 & 0xFF; own[1] = (o4 >> 8) & 0xFF; own[2] = (o4 >> 16) & 0xFF; own[3] = o4 >> 24;
        } else {
#pragma unroll
            for (int c = 0; c < 4; ++c) own[c] = c < n_valid ? occ[site0 + c] : 0xFFu;   // 0xFF never matches a row
        }
#pragma unroll
        for (int s = 0; s < 3; ++s) {
            if (s < P.S) {
                uint64_t h[4] = {0, 0, 0, 0};
                const int e0 = P.zoff[s], e1 = P.zoff[s + 1];
#pragma unroll 6
                for (int e = e0; e < e1; ++e) {
                    const int4 nb = __ldg(reinterpret_cast<const int4*>(P.nbr_slot + (size_t)e * P.Npad + site0));
                    h[0] += 1ull << (8 * occ[nb.x]);
                    h[1] += 1ull << (8 * occ[nb.y]);
                    h[2] += 1ull << (8 * occ[nb.z]);
                    h[3] += 1ull << (8 * occ[nb.w]);
                }
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const uint32_t hlo = (uint32_t)h[c], hhi = (uint32_t)(h[c] >> 32);
                    uint32_t e16[4];      // bytes spread into 16-bit fields: species (0,1) (2,3) (4,5) (6,7)
                    e16[0] = __byte_perm(hlo, 0, 0x4140);
                    e16[1] = __byte_perm(hlo, 0, 0x4342);
                    e16[2] = __byte_perm(hhi, 0, 0x4140);
                    e16[3] = __byte_perm(hhi, 0, 0x4342);
#pragma unroll
                    for (int i = 0; i < M; ++i) {
                        const bool mine = (own[c] == (uint32_t)i);
#pragma unroll
                        for (int w = 0; w < W; ++w) acc[s][i][w] += mine ? e16[w] : 0u;
                    }
                }
            }
        }
        since_flush += 4;
        if (since_flush >= kFlushSites) { flush(); since_flush = 0; }   // trip count is warp-uniform
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
// serial dependency chain and are applied by one thread (shared memory when the configuration fits, else global).
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
        if (threadIdx.x == 0) {
            for (int i = 0; i <= hi - lo; ++i) {
                const int n = hi - i;
                const uint32_t j = s_j[i];
                const uint8_t a = o[n], b = o[j];
                o[n] = b; o[j] = a;
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

// site-major [N][Z] -> slot-major [Z][Npad] (padding entries point at site 0)
__global__ void transpose_table_kernel(const int32_t* __restrict__ site_major, int32_t* __restrict__ slot_major,
                                       int N, int Npad, int Z)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (int64_t)Z * Npad) return;
    const int e = (int)(i / Npad), site = (int)(i % Npad);
    slot_major[i] = site < N ? site_major[(size_t)site * Z + e] : 0;
}

}  // namespace

// ---------------------------------------------------------------- launchers (called from hea_api.cu)
cudaError_t launch_sro_count(const KParams& P, const uint8_t* occ, int64_t B, int32_t* counts, int n_sms,
                             cudaStream_t st, int64_t* n_launches)
{
    const int SMM = P.S * P.M * P.M;
    cudaError_t e = cudaMemsetAsync(counts, 0, sizeof(int32_t) * (size_t)SMM * (size_t)B, st);
    if (e != cudaSuccess) return e;
    const int n_quads = P.Npad >> 2;
    int bx = (n_quads + kSroThreads - 1) / kSroThreads;
    // grid sized in multiples of the SM count: up to 8 resident blocks of 256 threads per SM
    const int64_t cap = (int64_t)n_sms * 8;
    int64_t want = cap / (B < 1 ? 1 : B);
    if (want < 1) want = 1;
    if (bx > want) bx = (int)want;
    for (int64_t b0 = 0; b0 < B; b0 += 65535) {
        const int by = (int)((B - b0) < 65535 ? (B - b0) : 65535);
        dim3 grid(bx, by);
        const uint8_t* o = occ + (size_t)b0 * P.N;
        int32_t* c = counts + (size_t)b0 * SMM;
        switch (P.M) {
            case 1: sro_count_kernel<1><<<grid, kSroThreads, 0, st>>>(P, o, c); break;
            case 2: sro_count_kernel<2><<<grid, kSroThreads, 0, st>>>(P, o, c); break;
            case 3: sro_count_kernel<3><<<grid, kSroThreads, 0, st>>>(P, o, c); break;
            case 4: sro_count_kernel<4><<<grid, kSroThreads, 0, st>>>(P, o, c); break;
            case 5: sro_count_kernel<5><<<grid, kSroThreads, 0, st>>>(P, o, c); break;
            case 6: sro_count_kernel<6><<<grid, kSroThreads, 0, st>>>(P, o, c); break;
            case 7: sro_count_kernel<7><<<grid, kSroThreads, 0, st>>>(P, o, c); break;
            default: sro_count_kernel<8><<<grid, kSroThreads, 0, st>>>(P, o, c); break;
        }
        ++*n_launches;
    }
    return cudaGetLastError();
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
                               const int64_t* n_per_species_dev, cudaStream_t st, int64_t* n_launches)
{
    const size_t base = kInitChunk * sizeof(uint32_t);
    const bool in_smem = (size_t)P.N + base <= 200 * 1024;
    cudaError_t e;
    if (in_smem) {
        const size_t smem = base + (size_t)P.N;
        e = cudaFuncSetAttribute(init_random_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        init_random_kernel<true><<<(unsigned)C, kInitThreads, smem, st>>>(P, occ, seed, chain0, n_per_species_dev);
    } else {
        init_random_kernel<false><<<(unsigned)C, kInitThreads, base, st>>>(P, occ, seed, chain0, n_per_species_dev);
    }
    ++*n_launches;
    return cudaGetLastError();
}

cudaError_t launch_stats_reset(void* stats, int64_t C, cudaStream_t st, int64_t* n_launches)
{
    stats_reset_kernel<<<(unsigned)((C + 255) / 256), 256, 0, st>>>(reinterpret_cast<uint64_t*>(stats), C);
    ++*n_launches;
    return cudaGetLastError();
}

cudaError_t launch_transpose_table(const int32_t* site_major, int32_t* slot_major, int N, int Npad, int Z,
                                   cudaStream_t st, int64_t* n_launches)
{
    const int64_t total = (int64_t)Z * Npad;
    transpose_table_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(site_major, slot_major, N, Npad, Z);
    ++*n_launches;
    return cudaGetLastError();
}

}  // namespace hea
