// hea_sro2.cu -- table-free ("stencil") full Warren-Cowley recount: the second engine behind hea_sro_full.
// DESIGN.md D4 and section 6.1b; Eq. 2, P:275 (the recount is >99% of the time of the
// non-incremental search); SURVEY 8(d) "recount, algorithmic minimum" / 8(f) f4.
//
// The table-driven kernel (hea_sro.cu) moves 4 Z + 1 bytes per atom and is bound by HBM.  On a regular lattice the
// neighbours need no table: this kernel moves ONE byte per atom and is bound by shared-memory loads and integer issue.
//   - a block walks a contiguous range of TILES of tx x ty x tz conventional cells.  It stages a tile plus a one-cell
//     halo (periodic images; every stencil shift is in {-1, 0, 1} cells) in shared memory, de-interleaved by basis
//     index, every site as a 32-bit word 1 << (FB * species), in a frame [basis][x][PY][PZ] whose pitches PY, PZ are
//     compile-time constants: a neighbour is then `LDS.32 [row pointer of its basis index + immediate]` plus one add
//     into a packed histogram, with no address arithmetic at all (the stencil is a constexpr table, checked against
//     the host builder's at launch);
//   - lanes run over the interior cells of a tile, z fastest (rows of tz <= 32 cells): where a warp spans two rows the
//     loads are 2-way bank-conflicted, which the LSU pipe (29 % busy) absorbs; the alternative mapping over the row words
//     INCLUDING the two halo words (conflict-free for every shape, tz / PZ of the lanes busy) is kept as `sro_lanes` = 1
//     and measured 9 % slower;
//   - HALF-SHELL: the shell vectors come in +-o pairs and the list of D2 is sorted, so the second half of every shell
//     is the negation of the first.  H_ij = #{(a, o in the positive half) : occ[a] = i, occ[a + o] = j} summed over all
//     sites gives the ordered pair counts as N_ij = H_ij + H_ji (re-index a' = a + o; holds for every cell size,
//     multi-edges and self-neighbours of tiny cells included).  Z/2 loads per site instead of Z;
//   - per site and shell the packed histogram h is split into NW words of wider fields and added to the per-thread row
//     of the site's own species under a predicate (no dynamic register indexing); rows are unpacked when the block
//     moves to another configuration (or the fields would overflow): warp REDUX, shared-memory bins, then one global
//     atomicAdd per bin with the transpose folded in.
// Integer adds commute: bit-exact with the table kernel and the oracle whatever the tiling.
#include <algorithm>
#include <atomic>
#include <utility>

#include "hea_device.cuh"
#include "hea_lattice.hpp"

namespace hea {

namespace {

constexpr int kStMaxThreads = 384;         // block size is chosen per tile shape (whole passes over the tile's words)
constexpr int kStPY = 10;                 // frame rows per x-plane: tiles are at most 8 cells along y
constexpr int kStMaxTx = 8;

// ---------------------------------------------------------------- the stencil as a compile-time table (D1-D2)
struct StEnt { int nb, sx, sy, sz; };

constexpr int kStD2[2][3] = {{2, 4, 6}, {3, 4, 8}};                       // squared shell radii in units of (a/2)^2
constexpr int kStZ[2][3] = {{12, 6, 24}, {8, 6, 12}};
constexpr int kStBasis[2][4][3] = {{{0, 0, 0}, {0, 1, 1}, {1, 0, 1}, {1, 1, 0}},
                                   {{0, 0, 0}, {1, 1, 1}, {0, 0, 0}, {0, 0, 0}}};

constexpr bool st_on_lattice(int lat, int x, int y, int z)
{
    return lat == 0 ? ((x + y + z) & 1) == 0 : ((x & 1) == (y & 1) && (y & 1) == (z & 1));
}

// Entry k (in the lexicographic order of D2) of shell s, seen from basis index b.
constexpr StEnt st_entry(int lat, int s, int k, int b)
{
    const int A = lat == 0 ? 4 : 2;
    int cnt = 0;
    for (int ox = -3; ox <= 3; ++ox)
        for (int oy = -3; oy <= 3; ++oy)
            for (int oz = -3; oz <= 3; ++oz) {
                if (ox * ox + oy * oy + oz * oz != kStD2[lat][s] || !st_on_lattice(lat, ox, oy, oz)) continue;
                if (cnt++ != k) continue;
                const int qx = kStBasis[lat][b][0] + ox, qy = kStBasis[lat][b][1] + oy, qz = kStBasis[lat][b][2] + oz;
                for (int nb = 0; nb < A; ++nb) {
                    const int dx = qx - kStBasis[lat][nb][0], dy = qy - kStBasis[lat][nb][1], dz = qz - kStBasis[lat][nb][2];
                    if ((dx & 1) == 0 && (dy & 1) == 0 && (dz & 1) == 0) return StEnt{nb, dx / 2, dy / 2, dz / 2};
                }
            }
    return StEnt{-1, 0, 0, 0};
}

// Half-shell entry E (0 .. ZH-1 over the concatenated positive halves) of basis index B in a frame of pitches PY, PZ.
template <int LAT, int PZ, int B, int E>
struct Nb {
    static constexpr int h0 = kStZ[LAT][0] / 2, h1 = kStZ[LAT][1] / 2;
    static constexpr int s = E < h0 ? 0 : (E < h0 + h1 ? 1 : 2);
    static constexpr int k = kStZ[LAT][s] / 2 + (E - (s == 0 ? 0 : (s == 1 ? h0 : h0 + h1)));
    static constexpr StEnt en = st_entry(LAT, s, k, B);
    static constexpr int nb = en.nb;
    static constexpr int imm = (en.sx * kStPY + en.sy) * PZ + en.sz;     // words, relative to the site's own slot
    static_assert(en.nb >= 0, "stencil entry not found");
};

// Packed histogram layout.  A site adds at most 12 per field and shell (half of z <= 24).
//   h    : species r is a field of FB bits at bit pos(r)                                  (one 32-bit word)
//   word : (h >> pos(w)) & MASK(w) -- species NW * f + w at bit FS * f                    (NW words, wider fields)
// MT <= 4: 8-bit fields -> 2 words x 2 fields of 16 bits.  MT = 8: 4-bit fields -> 4 words x 2 fields of 16 bits.
// MT = 5: 5-bit fields at bits 0, 5, 11, 16, 22 -> word 0 = species 0, 2, 4 in fields of 11, 11, 10 bits, word 1 =
// species 1, 3 in fields of 11 and 21 bits.
template <int MT>
struct Pack {
    static constexpr int FB = MT <= 4 ? 8 : (MT == 5 ? 5 : 4);
    static constexpr int NW = MT <= 4 ? 2 : (MT == 5 ? 2 : 4);
    static constexpr int FS = MT == 5 ? 11 : 16;                     // field spacing in the wide words
    static constexpr int kMinFieldBits = MT == 5 ? 10 : 16;
    static constexpr int kSitesCap = ((1 << kMinFieldBits) - 1) / 12;   // sites a lane may add before its rows are unpacked
    __host__ __device__ static constexpr int pos(int r) { return MT == 5 ? 5 * r + (r >> 1) : FB * r; }
    // pos() of four species bytes at once (species < 8: no carries between the bytes)
    __device__ __forceinline__ static uint32_t pos4(uint32_t v)
    {
        return MT == 5 ? v * 5u + ((v >> 1) & 0x7F7F7F7Fu) : v * (uint32_t)FB;
    }
    __host__ __device__ static constexpr uint32_t mask(int w)
    {
        uint32_t m = 0;
        for (int r = w; r < MT; r += NW) m |= ((1u << FB) - 1u) << (FS * (r / NW));
        return m;
    }
};

struct StencilParams {
    int tx, ty, tz;                       // tile extent, cells (tx <= 8, ty <= 8, tz <= PZ - 2)
    int ntx, nty, ntz;                    // tiles along x, y, z
    int plane;                            // words per basis index: (tx + 2) * PY * PZ
    int rows_load;                        // (ty + 2) * PZ: words staged per x-plane
    int rows_main;                        // ty * PZ: words the lanes run over per x-plane
    uint32_t mg_load, mg_main;            // magic of rows_load, rows_main
    int dense;                            // 1: lanes run over the interior cells only (rows of tz, 2-way bank conflicts
                                          // where a warp spans rows); 0: over the row words incl. the halo (conflict-free)
    uint32_t mg_tz, mg_ty;                // magic of tz, ty (dense mapping)
    int items_per_block;                  // contiguous (configuration, tile) items per block
    long long n_items;                    // B * tiles
    int cap_tiles;                        // tiles a lane may accumulate before unpacking its rows
};

// n / d = umulhi(2 n + 1, ceil(2^31 / d)) for n * d < 2^30 (d = 1 included)
__device__ __forceinline__ uint32_t div_magic(uint32_t n, uint32_t mg) { return __umulhi(2u * n + 1u, mg); }

template <int LAT, int PZ, int B, int E0, int... I>
__device__ __forceinline__ uint32_t shell_sum(const uint32_t* const (&bp)[4], std::integer_sequence<int, I...>)
{
    return (bp[Nb<LAT, PZ, B, E0 + I>::nb][Nb<LAT, PZ, B, E0 + I>::imm] + ...);
}

// One site of basis index B: Z/2 loads, S packed histograms, added to the rows of the site's own species.
template <int MT, int LAT, int S, int PZ, int B>
__device__ __forceinline__ void stencil_site(const uint32_t* const (&bp)[4], uint32_t (&acc)[S][MT][Pack<MT>::NW])
{
    using PK = Pack<MT>;
    constexpr int h0 = kStZ[LAT][0] / 2, h1 = kStZ[LAT][1] / 2, h2 = kStZ[LAT][2] / 2;
    const uint32_t own = bp[B][0];
    uint32_t h[S];
    h[0] = shell_sum<LAT, PZ, B, 0>(bp, std::make_integer_sequence<int, h0>{});
    if constexpr (S > 1) h[1] = shell_sum<LAT, PZ, B, h0>(bp, std::make_integer_sequence<int, h1>{});
    if constexpr (S > 2) h[2] = shell_sum<LAT, PZ, B, h0 + h1>(bp, std::make_integer_sequence<int, h2>{});
    // the row select is a multiply-add by the 0/1 flag "row r is mine": IMAD runs on the FMA pipe, which is otherwise
    // idle, instead of compare + select + add on the ALU pipe that already carries the histogram adds (ncu: ALU-bound)
    uint32_t mine[MT];
#pragma unroll
    for (int r = 0; r < MT; ++r) mine[r] = (own >> PK::pos(r)) & 1u;
#pragma unroll
    for (int s = 0; s < S; ++s)
#pragma unroll
        for (int w = 0; w < PK::NW; ++w) {
            const uint32_t word = (h[s] >> PK::pos(w)) & PK::mask(w);
#pragma unroll
            for (int r = 0; r < MT; ++r) acc[s][r][w] += word * mine[r];
        }
}

// MT = 4 serves M <= 4, MT = 5 serves M = 5, MT = 8 serves M = 6..8 (rows and fields >= M stay zero).
template <int MT, int LAT, int S, int PZ>
__global__ void __launch_bounds__(kStMaxThreads, 2)
sro_stencil_kernel(const KParams P, const StencilParams Q, const uint8_t* __restrict__ occ_all,
                   int32_t* __restrict__ counts_all)
{
    constexpr int A = LAT == 0 ? 4 : 2;
    constexpr int XP = kStPY * PZ;                                    // words per x-plane of the frame
    using PK = Pack<MT>;
    constexpr int NW = PK::NW, FS = PK::FS;
    constexpr int NB = S * MT * MT;

    extern __shared__ __align__(16) uint32_t s_w[];                   // [A][tx + 2][PY][PZ]
    __shared__ int s_bins[NB];
    for (int i = threadIdx.x; i < NB; i += blockDim.x) s_bins[i] = 0;

    const int M = P.M, SMM = S * M * M;
    const int Lx = P.L[0], Ly = P.L[1], Lz = P.L[2];
    const int n_tiles = Q.ntx * Q.nty * Q.ntz;
    const long long item0 = (long long)blockIdx.x * Q.items_per_block;
    const long long item1 = min(Q.n_items, item0 + (long long)Q.items_per_block);
    long long cfg = item0 / n_tiles;
    int tile = (int)(item0 - cfg * n_tiles);
    const int lane = threadIdx.x & 31;
    const int n_load = (Q.tx + 2) * Q.rows_load, n_main = Q.dense ? Q.tx * Q.ty * Q.tz : Q.tx * Q.rows_main;

    uint32_t acc[S][MT][NW];
#pragma unroll
    for (int s = 0; s < S; ++s)
#pragma unroll
        for (int r = 0; r < MT; ++r)
#pragma unroll
            for (int w = 0; w < NW; ++w) acc[s][r][w] = 0;
    int pending = 0;

    for (long long item = item0; item < item1; ++item) {
        int t = tile;
        const int tzi = t % Q.ntz; t /= Q.ntz;
        const int tyi = t % Q.nty;
        const int txi = t / Q.nty;
        const int x0 = txi * Q.tx, y0 = tyi * Q.ty, z0 = tzi * Q.tz;
        const uint8_t* __restrict__ occ = occ_all + (size_t)cfg * P.N;

        __syncthreads();                  // the previous tile has been read (first pass: the bins are zero)
        // ---- stage the tile and its halo: one padded cell (A sites) per thread and pass
        // (four cells in flight per thread: the global loads of a batch are issued before any of its stores; branch-free:
        // one conditional add / subtract wraps a coordinate because -1 <= g <= tiles * extent <= 2 L - 1)
        const uint32_t s_w_addr = (uint32_t)__cvta_generic_to_shared(s_w);
        const uint32_t plane_bytes = 4u * (uint32_t)Q.plane;
        for (int p0 = threadIdx.x; p0 < n_load; p0 += 4 * blockDim.x) {
            uint32_t v[4];
            int word[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int pu = p0 + u * blockDim.x;
                const bool in = pu < n_load;
                const int p = in ? pu : 0;
                const int px = (int)div_magic((uint32_t)p, Q.mg_load);
                const int r = p - px * Q.rows_load;
                const int py = r / PZ, pz = r - py * PZ;
                const bool use = in && pz <= Q.tz + 1;                // frame words beyond the tile's rows are not staged
                int gx = x0 + px - 1, gy = y0 + py - 1, gz = z0 + pz - 1;
                gx += gx < 0 ? Lx : 0;
                gx -= gx >= Lx ? Lx : 0;
                gy += gy < 0 ? Ly : 0;
                gy -= gy >= Ly ? Ly : 0;
                gz += gz < 0 ? Lz : 0;
                gz -= gz >= Lz ? Lz : 0;
                const int cell = (gx * Ly + gy) * Lz + gz;
                v[u] = 0;
                if (use) {
                    if (A == 4) v[u] = __ldg(reinterpret_cast<const uint32_t*>(occ) + cell);
                    else v[u] = __ldg(reinterpret_cast<const uint16_t*>(occ) + cell);
                }
                word[u] = use ? px * XP + r : -1;
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t p4 = PK::pos4(v[u]);                   // the bit positions of the cell's A species, bytewise
                const uint32_t dst = s_w_addr + 4u * (uint32_t)word[u];
#pragma unroll
                for (int b = 0; b < A; ++b) {
                    const uint32_t one = 1u << ((p4 >> (8 * b)) & 0xFFu);
                    if (word[u] >= 0) asm volatile("st.shared.u32 [%0], %1;" ::"r"(dst + (uint32_t)b * plane_bytes), "r"(one) : "memory");
                }
            }
        }
        __syncthreads();

        // ---- lanes run over the words of the interior rows; the halo words of a row idle
        for (int q = threadIdx.x; q < n_main; q += blockDim.x) {
            int x, r, y, pz;
            if (Q.dense) {
                const uint32_t q1 = div_magic((uint32_t)q, Q.mg_tz);
                pz = q - (int)q1 * Q.tz + 1;
                x = (int)div_magic(q1, Q.mg_ty);
                y = (int)q1 - x * Q.ty;
                r = y * PZ + pz;
            } else {
                x = (int)div_magic((uint32_t)q, Q.mg_main);
                r = q - x * Q.rows_main;
                y = r / PZ;
                pz = r - y * PZ;
            }
            if (pz < 1 || pz > Q.tz || x0 + x >= Lx || y0 + y >= Ly || z0 + pz - 1 >= Lz) continue;
            const uint32_t* bp[4];
#pragma unroll
            for (int b = 0; b < 4; ++b) bp[b] = s_w + (b < A ? b : 0) * Q.plane + (x + 1) * XP + PZ + r;
            stencil_site<MT, LAT, S, PZ, 0>(bp, acc);
            stencil_site<MT, LAT, S, PZ, 1>(bp, acc);
            if constexpr (A == 4) {
                stencil_site<MT, LAT, S, PZ, 2>(bp, acc);
                stencil_site<MT, LAT, S, PZ, 3>(bp, acc);
            }
        }

        ++pending;
        ++tile;
        const bool cfg_done = tile == n_tiles || item + 1 == item1;   // block-uniform
        if (cfg_done || pending == Q.cap_tiles) {
            // ---- unpack the rows: H[s][i][j] summed over the warp lands in lane k % 32, then one shared atomic per bin
            int mine[(NB + 31) / 32];
#pragma unroll
            for (int u = 0; u < (NB + 31) / 32; ++u) mine[u] = 0;
#pragma unroll
            for (int s = 0; s < S; ++s)
#pragma unroll
                for (int i = 0; i < MT; ++i)
#pragma unroll
                    for (int j = 0; j < MT; ++j) {
                        if (i >= M || j >= M) continue;
                        const int k = (s * MT + i) * MT + j;
                        const int v = (int)((acc[s][i][j % NW] >> (FS * (j / NW))) & ((1u << FS) - 1u));
                        const int tot = __reduce_add_sync(0xFFFFFFFFu, v);
                        if (lane == (k & 31)) mine[k >> 5] = tot;
                    }
#pragma unroll
            for (int u = 0; u < (NB + 31) / 32; ++u)
                if (lane + 32 * u < NB && mine[u]) atomicAdd(&s_bins[lane + 32 * u], mine[u]);
#pragma unroll
            for (int s = 0; s < S; ++s)
#pragma unroll
                for (int r = 0; r < MT; ++r)
#pragma unroll
                    for (int w = 0; w < NW; ++w) acc[s][r][w] = 0;
            pending = 0;
            if (cfg_done) {
                __syncthreads();
                // N_ij = H_ij + H_ji
                int32_t* counts = counts_all + (size_t)cfg * SMM;
                constexpr int NU = (NB + 127) / 128;                  // blocks have at least 128 threads
                int v[NU];
#pragma unroll
                for (int u = 0; u < NU; ++u) {
                    const int k = threadIdx.x + u * blockDim.x;
                    v[u] = 0;
                    if (k < SMM) {
                        const int s = k / (M * M), i = (k / M) % M, j = k % M;
                        v[u] = s_bins[(s * MT + i) * MT + j] + s_bins[(s * MT + j) * MT + i];
                        if (v[u]) atomicAdd(&counts[k], v[u]);
                    }
                }
                __syncthreads();
                for (int i = threadIdx.x; i < NB; i += blockDim.x) s_bins[i] = 0;
                if (tile == n_tiles) { tile = 0; ++cfg; }
            }
        }
    }
}

// Grid: a contiguous range of items per block, sized for the blocks that are resident at once (occupancy query x
// SMs, or blocks_per_sm if given), so that every block unpacks its rows as rarely as the item order allows.
template <int MT, int LAT, int S, int PZ>
cudaError_t launch_st_one(const KParams& P, StencilParams Q, const uint8_t* occ, int32_t* counts, int n_sms,
                          int blocks_per_sm, int threads, size_t smem, cudaStream_t st)
{
    auto kern = sro_stencil_kernel<MT, LAT, S, PZ>;
    // the shared-memory opt-in and the occupancy query are remembered per device for this instantiation (small launches
    // are latency-bound and would pay the two driver calls every time).  Each cache entry is ONE atomic word, so
    // concurrent callers read a consistent (threads, smem, resident) triple or repeat the driver call; a launch that
    // fails because the opt-in was lost (device reset, new primary context) opts in again and retries once, below.
    constexpr int kDevs = 16;
    static std::atomic<unsigned long long> s_optin[kDevs];
    static std::atomic<unsigned long long> s_occ[kDevs];      // threads (12 bits) | resident (12 bits) | smem (40 bits)
    cudaError_t e = cudaSuccess;
    int dev = 0;
    cudaGetDevice(&dev);
    const bool cached = dev >= 0 && dev < kDevs;
    if (!cached || smem > s_optin[dev].load(std::memory_order_acquire)) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (cached) s_optin[dev].store(smem, std::memory_order_release);
    }
    int resident = blocks_per_sm;
    if (resident <= 0) {
        const unsigned long long key = ((unsigned long long)threads & 0xFFFull) | ((unsigned long long)smem << 24);
        const unsigned long long got = cached ? s_occ[dev].load(std::memory_order_acquire) : 0ull;
        if (cached && (got & ~0xFFF000ull) == key && ((got >> 12) & 0xFFFull) != 0ull) resident = (int)((got >> 12) & 0xFFFull);
        else {
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, kern, threads, smem);
            if (e != cudaSuccess) return e;
            if (resident < 1) return cudaErrorInvalidConfiguration;
            if (cached) s_occ[dev].store(key | ((unsigned long long)(resident & 0xFFF) << 12), std::memory_order_release);
        }
    }
    const long long slots = (long long)n_sms * resident;
    long long ipb = (Q.n_items + slots - 1) / slots;
    ipb = std::max<long long>(1, std::min<long long>(ipb, 1 << 20));
    Q.items_per_block = (int)ipb;
    const long long grid = (Q.n_items + ipb - 1) / ipb;
    if (grid > 0x7FFFFFFF) return cudaErrorInvalidConfiguration;
    kern<<<(unsigned)grid, threads, smem, st>>>(P, Q, occ, counts);
    e = cudaGetLastError();
    if (e == cudaErrorInvalidValue && smem > 48u * 1024u) {
        // the cached opt-in no longer holds in this context: opt in again, retry once
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        kern<<<(unsigned)grid, threads, smem, st>>>(P, Q, occ, counts);
        e = cudaGetLastError();
    }
    return e;
}

template <int MT, int PZ>
cudaError_t launch_st_m(const KParams& P, const StencilParams& Q, int lat, const uint8_t* occ, int32_t* counts,
                        int n_sms, int blocks_per_sm, int threads, size_t smem, cudaStream_t st)
{
    switch (lat * 3 + P.S) {
        case 1: return launch_st_one<MT, 0, 1, PZ>(P, Q, occ, counts, n_sms, blocks_per_sm, threads, smem, st);
        case 2: return launch_st_one<MT, 0, 2, PZ>(P, Q, occ, counts, n_sms, blocks_per_sm, threads, smem, st);
        case 3: return launch_st_one<MT, 0, 3, PZ>(P, Q, occ, counts, n_sms, blocks_per_sm, threads, smem, st);
        case 4: return launch_st_one<MT, 1, 1, PZ>(P, Q, occ, counts, n_sms, blocks_per_sm, threads, smem, st);
        case 5: return launch_st_one<MT, 1, 2, PZ>(P, Q, occ, counts, n_sms, blocks_per_sm, threads, smem, st);
        default: return launch_st_one<MT, 1, 3, PZ>(P, Q, occ, counts, n_sms, blocks_per_sm, threads, smem, st);
    }
}

template <int PZ>
cudaError_t launch_st_pz(const KParams& P, const StencilParams& Q, int lat, const uint8_t* occ, int32_t* counts,
                         int n_sms, int blocks_per_sm, int threads, size_t smem, cudaStream_t st)
{
    if (P.M <= 4) return launch_st_m<4, PZ>(P, Q, lat, occ, counts, n_sms, blocks_per_sm, threads, smem, st);
    if (P.M == 5) return launch_st_m<5, PZ>(P, Q, lat, occ, counts, n_sms, blocks_per_sm, threads, smem, st);
    return launch_st_m<8, PZ>(P, Q, lat, occ, counts, n_sms, blocks_per_sm, threads, smem, st);
}

uint32_t magic_of(int d) { return (uint32_t)(((1ull << 31) + (uint64_t)d - 1) / (uint64_t)d); }

int split_even(int L, int cap, int* n_tiles)
{
    const int n = (L + cap - 1) / cap;
    *n_tiles = n;
    return (L + n - 1) / n;
}

constexpr int kStPZs[3] = {12, 22, 34};   // instantiated row pitches: tiles of up to 10, 20, 32 cells along z

}  // namespace

// The stencil engine reads a cell's A species as one word: occ (and occ + b * N, N = A * cells) must be A-aligned.
bool sro_stencil_usable(const Lattice& lat, const uint8_t* occ)
{
    return (reinterpret_cast<uintptr_t>(occ) % (uintptr_t)lat.A) == 0;
}

// tile_xy: cap on the tile extent along x and y, cells (0 = auto = 8, 1..8).  tile_z: row pitch variant (0 = auto: the
// one whose tiles fill the z extent best, else 12, 22 or 34).  lanes: 0/2 = interior cells, 1 = row words incl. halo.  blocks_per_sm: grid sizing (0 = auto: the occupancy query).
// opt_threads: block size (0 = auto, else a multiple of 32 in [128, 384]).
// flush_tiles: cap on the tiles a lane accumulates before its rows are unpacked (0 = auto: what the fields hold).
cudaError_t launch_sro_stencil(const KParams& P, const Lattice& lat, const uint8_t* occ, int64_t B, int32_t* counts,
                               int n_sms, int tile_xy, int tile_z, int blocks_per_sm, int flush_tiles, int opt_threads,
                               int lanes, cudaStream_t st,
                               int64_t* n_launches)
{
    const int SMM = P.S * P.M * P.M;
    cudaError_t e = cudaMemsetAsync(counts, 0, sizeof(int32_t) * (size_t)SMM * (size_t)B, st);
    if (e != cudaSuccess) return e;

    // the compile-time stencil must be the host builder's (D2): half-shell entry = second half of each sorted shell,
    // and its reverse is the mirrored entry of the neighbour's basis index.  Checked once per lattice type.
    static int s_checked[2] = {0, 0};                  // 0 = not yet, 1 = equal, -1 = differs (benign race: same value)
    if (s_checked[lat.type] == 0) {
        Lattice full;
        int ok = lattice_init(full, lat.type, 3, 3, 3, 3).empty() ? 1 : -1;
        for (int s = 0; ok == 1 && s < full.S; ++s) {
            if (full.z[s] != kStZ[full.type][s]) ok = -1;
            for (int k = 0; ok == 1 && k < full.z[s]; ++k)
                for (int b = 0; b < full.A; ++b) {
                    const StencilEntry& en = full.stencil[b][full.zoff[s] + k];
                    const StEnt ce = st_entry(full.type, s, k, b);
                    if (ce.nb != en.nb || ce.sx != en.sx || ce.sy != en.sy || ce.sz != en.sz) ok = -1;
                    const StencilEntry& rv = full.stencil[en.nb][full.zoff[s] + full.z[s] - 1 - k];
                    if (rv.nb != b || rv.sx != -en.sx || rv.sy != -en.sy || rv.sz != -en.sz) ok = -1;
                }
        }
        s_checked[lat.type] = ok;
    }
    if (s_checked[lat.type] != 1) return cudaErrorInvalidValue;

    int PZ = 0;
    if (tile_z > 0) PZ = tile_z;
    else {
        double best = -1.0;
        for (int v = 0; v < 3; ++v) {                  // best fill of the z extent of the tiles; ties: the longer rows
            const int cap = kStPZs[v] - 2, n = (lat.L[2] + cap - 1) / cap;
            const double fill = (double)lat.L[2] / ((double)n * cap);
            if (fill >= best - 1e-12) { best = std::max(best, fill); PZ = kStPZs[v]; }
        }
    }
    if (PZ != 12 && PZ != 22 && PZ != 34) return cudaErrorInvalidValue;

    StencilParams Q{};
    const int cap_xy = tile_xy > 0 ? std::min(tile_xy, kStMaxTx) : kStMaxTx;
    Q.tx = split_even(lat.L[0], cap_xy, &Q.ntx);
    Q.ty = split_even(lat.L[1], cap_xy, &Q.nty);
    Q.tz = split_even(lat.L[2], PZ - 2, &Q.ntz);
    Q.plane = (Q.tx + 2) * kStPY * PZ;
    Q.rows_load = (Q.ty + 2) * PZ;
    Q.rows_main = Q.ty * PZ;
    Q.mg_load = magic_of(Q.rows_load);
    Q.mg_main = magic_of(Q.rows_main);
    Q.dense = lanes == 1 ? 0 : 1;
    Q.mg_tz = magic_of(Q.tz);
    Q.mg_ty = magic_of(Q.ty);
    const int n_main = Q.dense ? Q.tx * Q.ty * Q.tz : Q.tx * Q.rows_main;
    // block size (measured on B200, profiles/r1_sweeps.md): small blocks when there are enough (configuration, tile)
    // items to fill the chip several times over -- six 4-warp blocks per SM overlap one block's staging with the
    // others' counting -- and larger blocks when a launch has few items, so that a tile is finished sooner.
    const int64_t n_items_all = (int64_t)Q.ntx * Q.nty * Q.ntz * B;
    int warps = n_items_all < n_sms ? 12 : (n_items_all < 5 * (int64_t)n_sms || PZ == 34 ? 8 : 4);
    if (opt_threads > 0) warps = opt_threads / 32;
    const int threads = warps * 32;
    const int sites_per_lane = ((n_main + threads - 1) / threads) * lat.A;
    const int sites_cap = P.M <= 4 ? Pack<4>::kSitesCap : (P.M == 5 ? Pack<5>::kSitesCap : Pack<8>::kSitesCap);
    Q.cap_tiles = std::max(1, sites_cap / sites_per_lane);
    if (sites_per_lane > sites_cap) return cudaErrorInvalidConfiguration;
    if (flush_tiles > 0) Q.cap_tiles = std::min(Q.cap_tiles, flush_tiles);
    const int64_t n_tiles = (int64_t)Q.ntx * Q.nty * Q.ntz;
    Q.n_items = (long long)(n_tiles * B);
    const size_t smem = sizeof(uint32_t) * (size_t)lat.A * Q.plane;
    switch (PZ) {
        case 12: e = launch_st_pz<12>(P, Q, lat.type, occ, counts, (unsigned)n_sms, blocks_per_sm, threads, smem, st); break;
        case 22: e = launch_st_pz<22>(P, Q, lat.type, occ, counts, (unsigned)n_sms, blocks_per_sm, threads, smem, st); break;
        default: e = launch_st_pz<34>(P, Q, lat.type, occ, counts, (unsigned)n_sms, blocks_per_sm, threads, smem, st); break;
    }
    if (e != cudaSuccess) return e;
    ++*n_launches;
    return cudaSuccess;
}

}  // namespace hea
