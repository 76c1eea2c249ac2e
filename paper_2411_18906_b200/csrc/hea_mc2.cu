// hea_mc2.cu -- chain-parallel Monte Carlo local search, second engine ("halo" engine) of hea_mc_run.
// DESIGN.md D6, D7, D9; Alg. 3, Eq. 4, Eq. 5, Eq. 6.
//
// Same algorithm, windows and results as hea_mc.cu (bit-exact trajectories); different data layout and gather:
//
//  * The chain's configuration lives in shared memory on a lattice PADDED by one ghost cell on every side
//    ((Lx+2)(Ly+2)(Lz+2) cells), ghosts holding the periodic images.  Every neighbour of every real site is then
//    `padded index + constant`, the constants depending only on the basis index of the site: no interior/boundary
//    distinction, no neighbour-table traffic in the kernel.  An accepted move also rewrites the ghost images (rare).
//  * A site is stored ONE-HOT (bit r = species r): a byte per site, or a nibble per site when M <= 4 and the bytes
//    do not fit (c4: 296,352 padded sites -> 148 KB).  A gather drops the loaded code into a byte slot of an
//    accumulator word (one IMAD); species counts of a shell come from (acc >> r) & 0x01010101 summed over the words
//    and one multiply by 0x01010101 -- no per-neighbour shift-by-species, no compare.
//  * Whether b is a neighbour of a (the exclusion of D9.2) comes from the lattice coordinates of the two sites
//    (minimum-image displacement, squared length == shell distance), not from a compare per table entry.
//  * Shell sizes and the basis count are template constants (fcc 12/6/24, bcc 8/6/12), so every gather is unrolled.
//
// Round 2: site decode by two exact multiply-high divisions, no coordinates; Philox round keys in
// kernel-parameter space; the first shell gathered without the offset table; the reject filter of long windows as an fp32
// quadratic form with a proven error bound in its threshold; the accept regime as a warp-specialised serial engine.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <type_traits>

#include "hea_device.cuh"
#include "hea_mc_common.cuh"

// The kernel is instantiated for 2 lattices x 2 selection rules x 8 species counts x 2 layouts x 2 target symmetries.
// To keep the build parallel, this file is compiled four times: HEA_MC2_PART = lattice + 2 * best-of-K (hea_mc2_p1..3.cu
// include it with the macro set); part 0 also holds the host-side dispatcher.
#ifndef HEA_MC2_PART
#define HEA_MC2_PART 0
#endif

namespace hea {

namespace {

enum { OCC2_U8 = 1, OCC2_NIB = 2 };

template <int LAT> struct LatC;
template <> struct LatC<0> { static constexpr int A = 4, lgA = 2, z0 = 12, z1 = 6, z2 = 24; };   // fcc
template <> struct LatC<1> { static constexpr int A = 2, lgA = 1, z0 = 8, z1 = 6, z2 = 12; };    // bcc
__host__ __device__ constexpr int pad4(int x) { return (x + 3) & ~3; }
template <int LAT> __host__ __device__ constexpr int zpad() { return pad4(LatC<LAT>::z0) + pad4(LatC<LAT>::z1) + pad4(LatC<LAT>::z2); }

// Lattice geometry of the padded layout (kernel parameter).
struct Geo {
    int L[3];
    uint32_t mq, sq;              // site / (A Lz)    = umulhi(site, mq) >> sq, exact for every site < 2^31 (see div_magic)
    uint32_t mx, sx;              // site / (A Ly Lz) = umulhi(site, mx) >> sx
    uint32_t cx, cc;              // padded index = site + 2 A q + cx x + cc,  q = site / (A Lz) = x Ly + y,  x = site / (A Ly Lz)
    uint32_t pmagy, pmagz;        // floor(2^32 / (Ly + 2)), floor(2^32 / (Lz + 2)): quotient off by <= 1 (load_state only)
    int PLy, PLz;                 // padded cell counts L + 2
    int NP;                       // padded sites
    uint32_t basis;               // bit 3b + d = doubled coordinate d of basis site b
    int d2[3];                    // squared shell distances in doubled units
    int distinct;                 // every L >= 3: a site pair is joined by at most one lattice vector of a shell
};

constexpr int kQueueCap = 1536;
constexpr int kDirty2Words = 1024;           // words of the hashed touched-site bitmap that lives in the queue
constexpr int kPaeK = 16;                   // pipelined accept engine: candidates per step evaluated ahead
constexpr int kPaeRecs = 512;               // records per epoch (= block threads): kPaeRecs / kPaeK steps

// A candidate evaluated ahead of its step (pipelined accept engine): everything that depends on the configuration but
// not on the pair counts.  Valid as long as none of its drawn sites was touched (or had a neighbour touched) since.
struct PRec {
    uint32_t a, b;                // the proposal after the redraw rule
    uint32_t a1, b1;              // the first draw (decides the redraw)
    uint32_t pqn;                 // p | q << 8 | null << 16 | absent << 17
    uint32_t pad;
    unsigned long long d0, d1, d2;   // Pack<M> species-count differences per shell, adjacency-corrected
};

struct Sh2 {
    int cnt[kSMM];
    double J;
    unsigned long long n_accept, n_null, hash, last_accept, n_logged;
    uint32_t best[3];
    uint32_t team_key;            // minimum key over the team (TEAM windows)
    unsigned long long bc_t0;     // follower: broadcast of the leader's phase record
    unsigned long long bc_depth;
    double bc_J;
    uint32_t bc_W, pad;
    MoveRec rec;
    // accept engine (8 lanes per candidate)
    MoveRec cand[32];             // improving records of the 32 groups of a round
    int4 wdesc[24];               // accumulator word w -> (int4 index in the offset row, slot mask, shell, side)
    uint4 mlog[kPaeRecs / kPaeK]; // serial accept engine: the move of each step of the epoch (a, b, p | q << 8 | 1 << 16, -)
    uint32_t swe_stop;            //   steps of the epoch consumed so far | (a step needs the candidates beyond kPaeK) << 31
    uint32_t sbest2[3];           //   lowest improving REBUILT record of a step (triple-buffered like sel)
    uint2 sel[3];                 //   (lowest improving record, mask of stale records) of a step
    double sJ[2][kPaeK];          //   J of the improving records of a step, by step parity (the role warps read one step behind)
    int4 fs_rd[4];                // first shell without the offset table: per basis index, per group of four, the part of a
                                  // neighbour's padded-index offset that depends on the site's basis (see Mc2Args::fs_c)
    double g[kSMM], t[kSMM];      // objective constants with a per-lane index
    // two-stage evaluation of long windows: integer pre-filter on shell 1, survivors queued for the full evaluation
    double nstar[64];             // first-shell cell (i, j): n*_ij = (1 - t_ij) / g_ij, the (real) count at which alpha = target
    double W1[64];                //                          w_1 g_ij^2
    uint32_t q_n[3];              // queue fill, triple-buffered like best[]
    uint32_t bestk;               // best-of-K: lowest key among the minimum-J candidates of the deciding step
    unsigned long long bestJ;     // best-of-K: minimum J (ordered_bits key) among the candidates of the deciding step
    uint32_t queue[kQueueCap];    // keys of the candidates that passed the pre-filter
};

struct SiteC {
    uint32_t pidx;                // padded site index
    int x, y, z, b;               // cell coordinates and basis index
};

// Site index -> cell coordinates, basis index and padded index.  Two exact multiply-high divisions by constants (a
// site index is divided by A Lz and by A Ly Lz directly, so no divisor is 1); the padded index needs no coordinates:
// ((x+1) PLy + (y+1)) PLz + (z+1) = cell + 2 q + 2 PLz x + (PLy PLz + PLz + 1) with q = x Ly + y.  y and z are dead code
// wherever only the padded index is used.
template <int LAT>
__device__ __forceinline__ SiteC decode_site(const Geo& G, uint32_t a)
{
    SiteC s;
    const uint32_t q = __umulhi(a, G.mq) >> G.sq;
    const uint32_t x = __umulhi(a, G.mx) >> G.sx;
    s.b = (int)(a & (uint32_t)(LatC<LAT>::A - 1));
    s.x = (int)x;
    s.y = (int)(q - x * (uint32_t)G.L[1]);
    s.z = (int)((a >> LatC<LAT>::lgA) - q * (uint32_t)G.L[2]);
    s.pidx = a + (uint32_t)(2 * LatC<LAT>::A) * q + G.cx * x + G.cc;
    return s;
}

template <int OCC>
__device__ __forceinline__ uint32_t occ_get(const uint8_t* s_occ, uint32_t pidx)
{
    if (OCC == OCC2_NIB) return ((uint32_t)s_occ[pidx >> 1] >> ((pidx & 1u) * 4u)) & 0xFu;
    return s_occ[pidx];
}

template <int OCC>
__device__ __forceinline__ void occ_set(uint8_t* s_occ, uint32_t pidx, uint32_t onehot)
{
    if (OCC == OCC2_NIB) {
        const uint32_t sh = (pidx & 1u) * 4u;
        s_occ[pidx >> 1] = (uint8_t)((s_occ[pidx >> 1] & ~(0xFu << sh)) | (onehot << sh));
    } else {
        s_occ[pidx] = (uint8_t)onehot;
    }
}

// Four loaded bytes (zero-extended) into the byte slots of a word: three multiply-adds, i.e. FMA-pipe instructions (the ALU
// pipe, which PRMT would use, is the busier one in the gather loops).
__device__ __forceinline__ uint32_t merge4(uint32_t x0, uint32_t x1, uint32_t x2, uint32_t x3)
{
    uint32_t lo, hi, w;
    asm("mad.lo.u32 %0, %1, 256, %2;" : "=r"(lo) : "r"(x1), "r"(x0));
    asm("mad.lo.u32 %0, %1, 256, %2;" : "=r"(hi) : "r"(x3), "r"(x2));
    asm("mad.lo.u32 %0, %1, 65536, %2;" : "=r"(w) : "r"(hi), "r"(lo));
    return w;
}

// One-hot codes of the ZS neighbours of a site in one shell, four byte slots per accumulator word.
// Table entries: OCC2_U8 -> padded index offset; OCC2_NIB -> 8 * byte offset + nibble shift, relative to the byte of the
// site.  The entries of a shell are ordered by the basis index of the neighbour (see the table build), so the four
// entries of a group share their nibble shift: four byte loads are merged into a word, then shifted and masked once.
template <int OCC, int ZS>
__device__ __forceinline__ void gather_shell(const uint8_t* __restrict__ s_occ, const int4* __restrict__ trow, uint32_t pidx,
                                             uint32_t (&acc)[(ZS + 3) / 4])
{
    const uint8_t* base = s_occ + (OCC == OCC2_NIB ? pidx >> 1 : pidx);
#pragma unroll
    for (int g = 0; g < (ZS + 3) / 4; ++g) {
        const int4 o = trow[g];
        uint32_t x[4] = {0u, 0u, 0u, 0u};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (g * 4 + j < ZS) {
                const int oj = j == 0 ? o.x : j == 1 ? o.y : j == 2 ? o.z : o.w;
                x[j] = base[OCC == OCC2_NIB ? (oj >> 3) : oj];
            }
        }
        uint32_t w = merge4(x[0], x[1], x[2], x[3]);
        if (OCC == OCC2_NIB) w = (w >> (o.x & 4)) & 0x0F0F0F0Fu;
        acc[g] = w;
    }
}

// First shell through Mc2Args::fs_c / fs_rd (no offset-table loads): same accumulator words as gather_shell, the groups
// being the odd-component classes of the lattice vectors.
template <int OCC, int NA>
__device__ __forceinline__ void gather_first_direct(const uint8_t* __restrict__ s_occ, const int4 rd, uint32_t pidx,
                                                    const int (&fc)[12], uint32_t (&acc)[NA])
{
#pragma unroll
    for (int g = 0; g < NA; ++g) {
        const uint32_t n = pidx + (uint32_t)(g == 0 ? rd.x : g == 1 ? rd.y : rd.z);
        const uint8_t* base = s_occ + (OCC == OCC2_NIB ? n >> 1 : n);
        const uint32_t x0 = base[fc[4 * g]], x1 = base[fc[4 * g + 1]], x2 = base[fc[4 * g + 2]], x3 = base[fc[4 * g + 3]];
        uint32_t w = merge4(x0, x1, x2, x3);
        if (OCC == OCC2_NIB) w = (w >> ((n & 1u) * 4u)) & 0x0F0F0F0Fu;
        acc[g] = w;
    }
}

// F[r] = #(neighbours of b of species r) - #(neighbours of a of species r) from the slot accumulators.
// Up to three words per site (shells of at most 12 neighbours): the one-hot bits of a byte are split into even and odd
// species, which leaves every species a 2-bit field, and the words of a site are ADDED before any per-species work.
template <int M, int NA>
__device__ __forceinline__ void hist_diff(const uint32_t (&accA)[NA], const uint32_t (&accB)[NA], int (&F)[M])
{
    int last = 0;
    if constexpr (NA <= 3) {
        uint32_t ea = 0, oa = 0, eb = 0, ob = 0;
#pragma unroll
        for (int g = 0; g < NA; ++g) {
            ea += accA[g] & 0x55555555u; oa += (accA[g] >> 1) & 0x55555555u;
            eb += accB[g] & 0x55555555u; ob += (accB[g] >> 1) & 0x55555555u;
        }
#pragma unroll
        for (int r = 0; r < M - 1; ++r) {
            const int sh = r & ~1;
            const uint32_t xa = ((r & 1 ? oa : ea) >> sh) & 0x03030303u, xb = ((r & 1 ? ob : eb) >> sh) & 0x03030303u;
            const uint32_t x = xb + (uint32_t)NA * 0x01010101u - xa;          // per byte in [0, 2 NA]
            F[r] = (int)((x * 0x01010101u) >> 24) - 4 * NA;
            last -= F[r];
        }
    } else {
#pragma unroll
        for (int r = 0; r < M - 1; ++r) {
            uint32_t x = (uint32_t)NA * 0x01010101u;             // per-byte bias: the byte sums stay in [0, 2 NA]
#pragma unroll
            for (int g = 0; g < NA; ++g) x += ((accB[g] >> r) & 0x01010101u) - ((accA[g] >> r) & 0x01010101u);
            F[r] = (int)((x * 0x01010101u) >> 24) - 4 * NA;
            last -= F[r];
        }
    }
    F[M - 1] = last;                                          // both sites have z_s entries: the differences sum to 0
}

// One shell's contribution in the D6 order, from the species-count differences F (see shell_sum in hea_mc_common.cuh).
template <int M, bool SYM>
__device__ __forceinline__ double shell_sum_F(const int* __restrict__ cnt, const double* __restrict__ g,
                                              const double* __restrict__ t, const int (&F)[M], const int (&c)[M])
{
    double up[M * M];
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

template <int M>
__device__ __forceinline__ typename Pack<M>::W pack_F(const int (&F)[M])
{
    typename Pack<M>::W d = 0;
#pragma unroll
    for (int r = 0; r < M; ++r) d |= (typename Pack<M>::W)(uint32_t)(F[r] + Pack<M>::kHalf) << (Pack<M>::FB * r);
    return d;
}

// ---- teams: R blocks per chain, synchronised through global memory (cooperative launch, all blocks co-resident)
//
// Few chains cannot fill 148 SMs with one block each, so a chain may be given a TEAM of R blocks, every block holding
// a replica of the chain state.  Windows run in one of two modes that all blocks of a team derive from the same
// history:
//   TEAM  the W*K candidates of the window are spread over the R*T threads; every block posts its best record into
//         its slot of the chain's control block and reads all R slots (release/acquire through L2), then every replica
//         applies the same move.  Worth its ~1-2 us exchange only when a window is several rounds of one block.
//   SOLO  block 0 (the leader) runs the windows alone -- in the accept regime a window is a fraction of one round and
//         extra blocks only add latency; the followers wait on the control block.  When the windows have grown, the
//         leader writes the state back, posts a phase record, and the followers reload and join.
constexpr int kMaxTeam = 32;
constexpr int kHaloThreads = 512;            // block size cap: 128 registers per thread, no spills in the hot paths
constexpr int kTeamRounds = 320;            // candidates per thread per window: longer windows amortise the imbalance between
                                            // warps and blocks at the window barrier, stage 2 and the team exchange (c4 reject regime,
                                            // trials/s, round 1: 32 rounds 3.9e10, 64 4.1e10, 128 4.25e10, 256 4.15e10; with the
                                            // site-histogram scan: 128 7.28e10, 192 7.55e10, 256 7.65e10, 320 7.74e10; 384 with 1,752 entries 7.80e10).  Bounded by the survivor
                                            // queue: 0.78 % of 320 x 512 candidates = 1,278 of its 1,536 entries (overflow: evaluated in place)
constexpr int kNullWords = kTeamRounds / 32; // 32-bit words of the per-thread null mask
// Reject-filter table: per ordered species pair (p, q) the elements threshold, X, L[M], Q[M], c'[M] (floats), stored
// element-major (element e of pair i at [e * M*M + i]) so that lanes with different pairs read different banks.
__host__ __device__ constexpr int filt_row(int M) { return 2 + 3 * M; }

struct TeamSlot {                 // 64 bytes
    uint32_t seq;                 // team-window number + 1 when the record below is valid
    uint32_t key, a, b, pq, pad;
    double J;
    uint64_t d[3];
};

struct TeamCtl {
    uint32_t phase_seq;           // number of phase records posted by the leader
    uint32_t W;                   // window length (steps) to continue with
    unsigned long long t0;        // next step
    double J;
    unsigned long long depth;     // search-depth counter (hea_mc_run_ex)
    uint32_t hist_bar;            // arrivals at the team barrier that ends a site-histogram build (monotone)
    uint32_t pad[7];
    TeamSlot slot[2][kMaxTeam];   // [team-window parity][rank]
};

__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p)
{
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void st_release_u32(uint32_t* p, uint32_t v)
{
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

struct Mc2Args {
    McArgs a;                     // a.R = blocks per chain
    Geo G;
    TeamCtl* team;                // [C] control blocks, zeroed before the launch (R > 1 only)
    int team_on, team_off;        // enter TEAM when W*K >= team_on; leave it after a move with steps_done*K < team_off
    int accept_engine;            // 1: single-step windows run on the 8-lanes-per-candidate engine
    int pae;                      // 1: ... pipelined over epochs of steps (record, dirty-bitmap and offset buffers present)
    int dshift;                   //    log2 of the sites per bit of its touched-site bitmap
    double filt_floor;            // reject filter: absolute floor of its threshold
    uint32_t* hist;               // [C][N] site-histogram table of the reject filter, or nullptr: per site
                                  // species << 24 | first-shell neighbour counts of species 0..M-2 in fields of 8 (M <= 4) or
                                  // 6 (M = 5) bits; read and written through L2 only
    uint32_t k_mq, k_sq;          // candidate index / K = umulhi(index, k_mq) >> k_sq (K >= 2)
    uint32_t rk[20];              // Philox round keys of the seed (D7): key + r * (0x9E3779B9, 0xBB67AE85), r = 0..9
    // First shell without the offset table.  A first-shell lattice vector v reaches, from basis offset beta (components
    // 0/1), the cell shifted by floor(v_d / 2) + beta_d [v_d odd]: the padded-index offset splits into a part that depends
    // only on v (fs_c: A * cell part, same for every site; stored halved for the nibble layout) and a part that depends
    // only on the site's basis index and on WHICH components of v are odd (fs_rd[b][group]; the vectors are grouped by
    // that pattern, four per group).  neighbour = pidx + fs_rd[b][g] + fs_c[g][j]: one add with a constant-bank operand.
    int fs_c[12];
    int fs_rd[4][4];
    // hea_mc_run_ex
    int select_best;              // 1: the minimum J_k of a step is taken (ties -> lowest k) instead of the lowest improving k
    unsigned long long depth_limit;        // > 0: a chain stops after this many consecutive steps without a move
    unsigned long long* depth_all;         // [C] in/out, or nullptr
    unsigned long long* steps_done_all;    // [C] out, or nullptr
};

// ---- stage 1 of a long window from the site-histogram table
constexpr int kHistBatch = 4;     // candidates a thread keeps in flight
struct HistArgs {                 // the same in every thread of the block
    const uint32_t* H;            // the chain's table: species << 24 | first-shell neighbour counts of species 0..M-2
    const uint32_t* rk;           // Philox round keys (Mc2Args::rk)
    // shared-memory objects as 32-bit shared-space addresses (a generic pointer would make every access a generic LD / ATOM)
    uint32_t best_slot;           // lowest improving key found so far in this window
    uint32_t ftab;                // reject-filter table, element-major
    uint32_t queue;               // keys of the survivors
    uint32_t q_n;
    unsigned long long t0;        // first step of the window
    uint32_t Wc, ts_inc, k_inc, K, N, chain;
    int Lx, Ly, Lz;
    uint32_t mx, sx, mq, sq;      // site / (A Ly Lz), site / (A Lz) by multiply-high (Geo)
    uint32_t cx, cc;              // padded index = site + 2 A q + cx x + cc (Geo)
    uint32_t occ;                 // shared-space address of the padded one-hot configuration
    uint32_t basis;
    int d2_0;                     // squared first-shell distance, doubled units
};

struct HistScan {                 // one thread's scan of its candidates of the window
    uint32_t ts, k;               // next candidate (window step, k)
    uint32_t ncur;                // null bits of the current group of 32 candidates
    int j;                        // candidates scanned
    uint32_t nullw[kNullWords];
    uint32_t ovf[kTeamRounds];    // survivors that found the queue full: the caller evaluates them
    int n_ovf;
    int done;
};

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t lds_volatile_u32(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t lds_u8(uint32_t a)
{
    uint32_t v;
    asm("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ float lds_f32(uint32_t a)
{
    float v;
    asm("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t atoms_inc(uint32_t a)
{
    uint32_t v;
    asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u32(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }

// Scans this thread's candidates in batches of four: Philox, the species of the drawn sites from the configuration in shared
// memory (which settles redraw and nullness, D9.1), the two table words of a live candidate (its only L2 round trip),
// first-shell adjacency (D9.2), F = difference of the neighbour counts, the fp32 form of the reject filter; survivors go
// to the queue.  What bounds it is the rate at which an SM takes random 32-byte sectors from L2 (~0.75 per clock with the
// 196 KB carve-out, measured), hence as few loads per candidate as possible.  Not inlined on purpose: inside the kernel body the loop would share 128 registers with everything else
// that is live there, and the allocator then reuses load destinations, which serialises the L2 round trips.
template <int M, int LAT, bool BEST, int OCC>
__device__ __noinline__ void hist_scan(HistScan& st, const HistArgs& A)
{
    constexpr int U = kHistBatch;
    static_assert(32 % U == 0, "null words are closed on batch boundaries");
    constexpr int MM = M * M;
    constexpr int HFB = M <= 4 ? 8 : 6;
    constexpr uint32_t HFM = (1u << HFB) - 1u;
    constexpr uint32_t kBias = (M > 1 ? 16u : 0u) | (M > 2 ? 16u << HFB : 0u) | (M > 3 ? 16u << (2 * HFB) : 0u) |
                               (M > 4 ? 16u << (3 * HFB) : 0u);
    using LC = LatC<LAT>;
    uint32_t rk[20];
#pragma unroll
    for (int i = 0; i < 20; ++i) rk[i] = A.rk[i];
    const uint32_t* __restrict__ H = A.H;
    const uint32_t N = A.N, K = A.K, Wc = A.Wc, ts_inc = A.ts_inc, k_inc = A.k_inc, chain = A.chain;
    const unsigned long long t0 = A.t0;
    const int Lx = A.Lx, Ly = A.Ly, Lz = A.Lz;
    const uint32_t Lxy = (uint32_t)(Lx * Ly);
    const uint32_t mx = A.mx, sx = A.sx, mq = A.mq, sq = A.sq, gcx = A.cx, gcc = A.cc, occ_s = A.occ;
    // one-hot species code of the site with cell-row index q = x Ly + y and x, from the padded configuration in shared memory
    auto code_at = [&](uint32_t site, uint32_t q, uint32_t x) -> uint32_t {
        const uint32_t pidx = site + (uint32_t)(2 * LC::A) * q + gcx * x + gcc;
        if (OCC == OCC2_NIB) return (lds_u8(occ_s + (pidx >> 1)) >> ((pidx & 1u) * 4u)) & 0xFu;
        return lds_u8(occ_s + pidx);
    };
    uint32_t ts = st.ts, k = st.k, ncur = 0u;
    int j = 0, n_ovf = 0;
    while (ts < Wc) {
        const uint32_t hint = lds_volatile_u32(A.best_slot);
        if ((hint >> 10) < ts) break;                               // a move at an earlier step exists
        uint32_t key[U], a[U], b[U], ha[U], hb[U], qa[U], qb[U];
        int cx[U];
        bool live[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            key[u] = ts < Wc ? ((ts << 10) | k) : kNoKey;
            const unsigned long long step = t0 + ts;
            const uint4 r = philox4x32_10_rk((uint32_t)step, (uint32_t)(step >> 32), k, chain, rk);
            // D9.1.  The cell coordinates of a come straight from its random word: floor(floor(r N / 2^32) / d) =
            // floor(r (N / d) / 2^32); those of b by the exact multiply-high divisions of Geo.
            uint32_t sa = __umulhi(r.x, N), sb = __umulhi(r.y, N - 1u);
            sb += (sb >= sa);
            uint32_t xa = __umulhi(r.x, (uint32_t)Lx), ya = __umulhi(r.x, Lxy);
            uint32_t xb = __umulhi(sb, mx) >> sx, yb = __umulhi(sb, mq) >> sq;
            uint32_t ca = code_at(sa, ya, xa), cb = code_at(sb, yb, xb);
            if (ca == cb) {                                         // like species: redraw once
                sa = __umulhi(r.z, N); sb = __umulhi(r.w, N - 1u);
                sb += (sb >= sa);
                xa = __umulhi(r.z, (uint32_t)Lx); ya = __umulhi(r.z, Lxy);
                xb = __umulhi(sb, mx) >> sx; yb = __umulhi(sb, mq) >> sq;
                ca = code_at(sa, ya, xa); cb = code_at(sb, yb, xb);
            }
            live[u] = ca != cb;
            a[u] = sa; b[u] = sb; qa[u] = ya; qb[u] = yb; cx[u] = (int)xb - (int)xa;
            ha[u] = 0u; hb[u] = 0u;
            if (live[u]) { ha[u] = __ldcg(H + sa); hb[u] = __ldcg(H + sb); }     // the only L2 round trip of a candidate
            k += k_inc; ts += ts_inc;
            if (k >= K) { k -= K; ++ts; }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            ncur = __funnelshift_r(ncur, live[u] ? 0u : 1u, 1);
            if (live[u] && key[u] != kNoKey && (BEST || key[u] < hint)) {
                const int p = (int)(ha[u] >> 24), q = (int)(hb[u] >> 24);
                // D9.2: are a and b first-shell neighbours?  Almost every pair fails on x or y.
                const int cy = (int)(qb[u] - qa[u]) - cx[u] * Ly;
                const int ax = abs(cx[u]), ay = abs(cy);
                int mm0 = 0;
                if ((ax <= 1 || ax == Lx - 1) && (ay <= 1 || ay == Ly - 1)) {
                    const uint32_t sa = a[u], sb = b[u];
                    const int za = (int)((sa >> LC::lgA) - qa[u] * (uint32_t)Lz), zb = (int)((sb >> LC::lgA) - qb[u] * (uint32_t)Lz);
                    const int ba = (int)(sa & (uint32_t)(LC::A - 1)), bb = (int)(sb & (uint32_t)(LC::A - 1));
                    const int dx = 2 * cx[u] + (int)((A.basis >> (3 * bb)) & 1u) - (int)((A.basis >> (3 * ba)) & 1u);
                    const int dy = 2 * cy + (int)((A.basis >> (3 * bb + 1)) & 1u) - (int)((A.basis >> (3 * ba + 1)) & 1u);
                    const int dz = 2 * (zb - za) + (int)((A.basis >> (3 * bb + 2)) & 1u) - (int)((A.basis >> (3 * ba + 2)) & 1u);
                    const int wx = dx > Lx ? dx - 2 * Lx : dx < -Lx ? dx + 2 * Lx : dx;
                    const int wy = dy > Ly ? dy - 2 * Ly : dy < -Ly ? dy + 2 * Ly : dy;
                    const int wz = dz > Lz ? dz - 2 * Lz : dz < -Lz ? dz + 2 * Lz : dz;
                    mm0 = (wx * wx + wy * wy + wz * wz) == A.d2_0;
                }
                const uint32_t X = (hb[u] & 0xFFFFFFu) + kBias - (ha[u] & 0xFFFFFFu);      // fields in [4, 28]: no borrow
                int F0[M];
                int last = 0;
#pragma unroll
                for (int r2 = 0; r2 < M - 1; ++r2) {
                    F0[r2] = (int)((X >> (HFB * r2)) & HFM) - 16;
                    last -= F0[r2];
                }
                F0[M - 1] = last;
                if (mm0 != 0) {
#pragma unroll
                    for (int r2 = 0; r2 < M; ++r2) F0[r2] -= (r2 == p) - (r2 == q);
                }
                const uint32_t row = A.ftab + 4u * (uint32_t)(p * M + q);       // element e at row + 4 e MM
                float acc = 0.0f, D = 0.0f;
#pragma unroll
                for (int r2 = 0; r2 < M; ++r2) {
                    const float f = (float)F0[r2];
                    acc = fmaf(fmaf(lds_f32(row + 4u * (2 + M + r2) * MM), f, lds_f32(row + 4u * (2 + r2) * MM)), f, acc);
                    D = fmaf(lds_f32(row + 4u * (2 + 2 * M + r2) * MM), f, D);
                }
                acc = fmaf(lds_f32(row + 4u * MM) * D, D, acc);
                if (!(acc > lds_f32(row))) {
                    const uint32_t slot = atoms_inc(A.q_n);
                    if (slot < (uint32_t)kQueueCap) sts_u32(A.queue + 4u * slot, key[u]);
                    else st.ovf[n_ovf++] = key[u];                 // at most kTeamRounds candidates per thread and window
                }
            }
        }
        j += U;
        if ((j & 31) == 0) st.nullw[(j >> 5) - 1] = ncur;
    }
    st.ts = ts; st.k = k; st.ncur = ncur; st.j = j; st.n_ovf = n_ovf; st.done = 1;
}

// Shared memory: occupancy (offset 0, so a gather address is the loaded offset itself) | Sh2 | offset table [A][ZP].
template <int M, int OCC, bool SYM, int LAT, bool BEST>
__global__ void __launch_bounds__(kHaloThreads)
mc_halo_kernel(const KParams P, const __grid_constant__ McConst<M> Kc, const __grid_constant__ Mc2Args AA)
{
    extern __shared__ __align__(16) uint8_t s_raw[];
    using LC = LatC<LAT>;
    constexpr int ZP = zpad<LAT>();
    constexpr int NA0 = (LC::z0 + 3) / 4, NA1 = (LC::z1 + 3) / 4, NA2 = (LC::z2 + 3) / 4;
    constexpr int MM = M * M;
    using PW = typename Pack<M>::W;
    const McArgs& A = AA.a;
    const Geo& G = AA.G;
    const uint32_t occ_bytes = (uint32_t)(((OCC == OCC2_NIB ? (G.NP + 1) / 2 : G.NP) + 15) & ~15);
    uint8_t* s_occ = s_raw;
    Sh2& sh = *reinterpret_cast<Sh2*>(s_raw + occ_bytes);
    int* s_tab = reinterpret_cast<int*>(s_raw + occ_bytes + ((sizeof(Sh2) + 15) & ~(size_t)15));
    // pipelined accept engine buffers (only when AA.pae): records | dirty bitmap over logical sites | logical offsets [A][Z]
    constexpr int RS = filt_row(M);
    float* s_ftab = reinterpret_cast<float*>(s_tab + LC::A * ZP);       // [RS][M*M] reject-filter table, element-major
    PRec* s_prec = reinterpret_cast<PRec*>(s_ftab + ((MM * RS + 3) & ~3));
    uint32_t* s_dirty = reinterpret_cast<uint32_t*>(s_prec + kPaeRecs);
    // one bit per group of 2^dshift consecutive sites (coarser = conservative: more records count as stale)
    const uint32_t dshift = (uint32_t)AA.dshift;
    const int dwords = (int)(((((uint32_t)P.N + (1u << dshift) - 1u) >> dshift) + 31u) >> 5);
    int* s_loff = reinterpret_cast<int*>(s_dirty + dwords);
    // second, hashed view of the same touched set: bit (site mod 32 kDirty2Words), in the first words of the survivor queue (which is
    // idle while the serial accept engine runs).  A site counts as touched only when BOTH bitmaps say so: the coarse one
    // flags whole groups of 2^dshift neighbouring sites, this one separates them again (conservative: no false negative).
    uint32_t* const s_dirty2 = sh.queue;
    bool mark2 = false;                                      // inside a serial-engine epoch (block-uniform)
    auto mark_bits = [&](uint32_t v) {
        atomicOr(&s_dirty[v >> (5u + dshift)], 1u << ((v >> dshift) & 31u));
        if (mark2) atomicOr(&s_dirty2[(v >> 5) & (uint32_t)(kDirty2Words - 1)], 1u << (v & 31u));
    };
    auto touched = [&](uint32_t v) -> uint32_t {
        return (s_dirty[v >> (5u + dshift)] >> ((v >> dshift) & 31u)) & (s_dirty2[(v >> 5) & (uint32_t)(kDirty2Words - 1)] >> (v & 31u)) & 1u;
    };
    // serial accept engine: packed count changes per objective row of the improving records, [step parity][record][S*M]
    // (8-byte aligned through its byte offset from s_raw, not through an integer cast of the pointer: the compiler then
    // keeps the shared address space and emits LDS / STS instead of generic loads and stores for s_dn and s_px)
    unsigned long long* s_dn = reinterpret_cast<unsigned long long*>(
        s_raw + (((size_t)(reinterpret_cast<uint8_t*>(s_loff + LC::A * P.Z) - s_raw) + 7u) & ~(size_t)7u));
    // per record: padded index of a and of b, bit 31 = the site's cell is interior (no ghost image, neighbours = site + offset)
    uint2* s_px = reinterpret_cast<uint2*>(s_dn + 2 * kPaeK * P.S * P.M);

    const int tid = threadIdx.x, T = blockDim.x;
    const int S = P.S, N = P.N, K = A.K, R = A.R;
    const int SMM = S * MM;
    const uint32_t rank = R > 1 ? blockIdx.x % (unsigned)R : 0u;
    const size_t chain_local = R > 1 ? blockIdx.x / (unsigned)R : blockIdx.x;
    uint8_t* g_occ = A.occ_all + chain_local * (size_t)N;
    int32_t* g_cnt = A.counts_all + chain_local * (size_t)SMM;
    unsigned long long* g_stats = A.stats_all + chain_local * 5;
    TeamCtl* ctl = R > 1 ? AA.team + chain_local : nullptr;
    const uint32_t chain = (uint32_t)(A.chain0 + chain_local);
    const int Lx = G.L[0], Ly = G.L[1], Lz = G.L[2];

    // counts and the padded one-hot configuration from global memory (L2 loads: a leader may just have written them)
    auto load_state = [&]() {
        for (int i = tid; i < SMM; i += T) sh.cnt[i] = __ldcg(g_cnt + i);
        auto code_of = [&](int pi) -> uint32_t {           // one-hot code of padded site pi (ghosts = periodic images)
            if (pi >= G.NP) return 0u;
            const int b = pi & (LC::A - 1);
            const uint32_t cell = (uint32_t)pi >> LC::lgA;
            uint32_t q1 = __umulhi(cell, G.pmagz);
            int pz = (int)(cell - q1 * (uint32_t)G.PLz);
            if (pz >= G.PLz) { pz -= G.PLz; ++q1; }
            uint32_t q2 = __umulhi(q1, G.pmagy);
            int py = (int)(q1 - q2 * (uint32_t)G.PLy);
            if (py >= G.PLy) { py -= G.PLy; ++q2; }
            const int px = (int)q2;
            const int x = px == 0 ? Lx - 1 : px == Lx + 1 ? 0 : px - 1;
            const int y = py == 0 ? Ly - 1 : py == Ly + 1 ? 0 : py - 1;
            const int z = pz == 0 ? Lz - 1 : pz == Lz + 1 ? 0 : pz - 1;
            const int site = (((x * Ly + y) * Lz + z) << LC::lgA) | b;
            return 1u << __ldcg(g_occ + site);
        };
        if (OCC == OCC2_NIB) {
            for (int i = tid; i < (G.NP + 1) / 2; i += T) s_occ[i] = (uint8_t)(code_of(2 * i) | (code_of(2 * i + 1) << 4));
        } else {
            for (int i = tid; i < G.NP; i += T) s_occ[i] = (uint8_t)code_of(i);
        }
    };
    auto store_state = [&]() {
        for (int i = tid; i < N; i += T) {
            const SiteC sc = decode_site<LAT>(G, (uint32_t)i);
            g_occ[i] = (uint8_t)(31 - __clz((int)occ_get<OCC>(s_occ, sc.pidx)));
        }
        for (int i = tid; i < SMM; i += T) g_cnt[i] = sh.cnt[i];
    };

    // ---- prologue
    load_state();
    for (int i = tid; i < LC::A * ZP; i += T) {
        const int b = i / ZP, slot = i - b * ZP;
        int s, e;
        if (slot < pad4(LC::z0)) { s = 0; e = slot; }
        else if (slot < pad4(LC::z0) + pad4(LC::z1)) { s = 1; e = slot - pad4(LC::z0); }
        else { s = 2; e = slot - pad4(LC::z0) - pad4(LC::z1); }
        const int zs = s == 0 ? LC::z0 : s == 1 ? LC::z1 : LC::z2;
        int entry = 0;
        if (s < S && e < zs) {
            // slot e holds the entry that comes e-th when the shell is ordered by the neighbour's basis index
            const int8_t* st = P.tab->stencil + (b * P.Z + (int)P.tab->by_basis[b * P.Z + P.zoff[s] + e]) * 4;     // (nb, sx, sy, sz)
            const int off = ((((int)st[1] * G.PLy + (int)st[2]) * G.PLz + (int)st[3]) << LC::lgA) + ((int)st[0] - b);
            if (OCC == OCC2_NIB) {
                const int tt = (b & 1) + off;                 // padded index parity of the site == b & 1 (A is even)
                entry = (tt >> 1) * 8 + (tt & 1) * 4;         // byte offset * 8 + nibble shift
            } else {
                entry = off;
            }
        }
        s_tab[i] = entry;
    }
    for (int i = tid; i < SMM; i += T) { sh.g[i] = Kc.g[i]; sh.t[i] = Kc.t[i]; }
    if (tid < 4) sh.fs_rd[tid] = make_int4(AA.fs_rd[tid][0], AA.fs_rd[tid][1], AA.fs_rd[tid][2], AA.fs_rd[tid][3]);
    for (int i = tid; i < MM; i += T) {
        const double gi = Kc.g[i];
        sh.nstar[i] = (1.0 - Kc.t[i]) / gi;
        sh.W1[i] = Kc.w[0] * gi * gi;
    }
    if (AA.pae) {
        for (int i = tid; i < dwords; i += T) s_dirty[i] = 0u;
        for (int i = tid; i < LC::A * P.Z; i += T) {      // neighbour e of a site of basis b without periodic wrap
            const int8_t* st = P.tab->stencil + i * 4;
            const int b = i / P.Z;
            s_loff[i] = ((((int)st[1] * Ly + (int)st[2]) * Lz + (int)st[3]) << LC::lgA) + ((int)st[0] - b);
        }
    }
    if (tid < 24) {
        // word list of the accept engine: per shell s < S the NA_s words of site a, then the NA_s words of site b
        int w = tid, s = 0, side = 0, g = 0, rowoff = 0;
        bool ok = false;
        for (int s2 = 0, w0 = 0, ro = 0; s2 < S; ++s2) {
            const int na = s2 == 0 ? NA0 : s2 == 1 ? NA1 : NA2;
            if (w >= w0 && w < w0 + 2 * na) { ok = true; s = s2; side = (w - w0) >= na; g = (w - w0) - side * na; rowoff = ro; }
            w0 += 2 * na; ro += na;
        }
        const int zs = s == 0 ? LC::z0 : s == 1 ? LC::z1 : LC::z2;
        const int valid = ok ? min(4, zs - 4 * g) : 0;
        const uint32_t mask = valid >= 4 ? 0xFFFFFFFFu : ((1u << (8 * valid)) - 1u);
        sh.wdesc[tid] = make_int4(rowoff + g, (int)mask, s, side);
    }
    if (tid == 0) {
        sh.n_accept = g_stats[0]; sh.n_null = 0; sh.hash = g_stats[2]; sh.last_accept = g_stats[3]; sh.n_logged = 0;
        sh.best[0] = sh.best[1] = sh.best[2] = kNoKey;
        sh.q_n[0] = sh.q_n[1] = sh.q_n[2] = 0u;
        sh.bestk = kNoKey; sh.bestJ = ~0ull;
        sh.rec.key = kNoKey;
    }
    __syncthreads();
    if (tid == 0) {
        double J = 0.0;
        for (int s = 0; s < S; ++s)
            J = __dadd_rn(J, __dmul_rn(Kc.w[s], shell_sum<M, false>(sh.cnt + s * MM, Kc.g + s * MM, Kc.t + s * MM, Pack<M>::bias(), 0, 0)));
        sh.J = J;
    }
    __syncthreads();

    const int32_t* __restrict__ nbr = P.nbr_site;
    const bool prune = A.prune != 0;

    // candidate c of a window (ordered by (step, k)) belongs to thread gtid = c mod GT; GT depends on the mode
    bool team = false;                                       // every chain starts SOLO with W = 1
    uint32_t GT, gtid, ts_first, k_first, ts_inc, k_inc, w_cap;
    auto set_mode = [&](bool tm) {
        team = tm;
        GT = tm ? (uint32_t)T * (uint32_t)R : (uint32_t)T;
        gtid = tm ? (uint32_t)tid * (uint32_t)R + rank : (uint32_t)tid;
        ts_first = gtid / (uint32_t)K; k_first = gtid - ts_first * (uint32_t)K;
        ts_inc = GT / (uint32_t)K; k_inc = GT - ts_inc * (uint32_t)K;
        w_cap = (uint32_t)min((uint64_t)(1u << 20), ((uint64_t)kTeamRounds * GT) / (uint32_t)K);
        if (w_cap < 1u) w_cap = 1u;
        if (w_cap > (uint32_t)A.w_max) w_cap = (uint32_t)A.w_max;
    };
    set_mode(false);
    constexpr bool best_mode = BEST;
    const unsigned long long depth_limit = AA.depth_limit;
    unsigned long long depth = (depth_limit && AA.depth_all) ? AA.depth_all[chain_local] : 0ull;
    const bool accept_ok = T >= 512 && AA.accept_engine != 0 && !best_mode;   // 8 evaluating warps + null-settling warps

    // one-hot code of a site and of its ghost images (only cells on the boundary have any)
    auto write_site = [&](uint32_t u, uint32_t code) {
        const SiteC sc = decode_site<LAT>(G, u);
        if (sc.x >= 1 && sc.x <= Lx - 2 && sc.y >= 1 && sc.y <= Ly - 2 && sc.z >= 1 && sc.z <= Lz - 2) {
            occ_set<OCC>(s_occ, sc.pidx, code);               // interior cell: no ghost image
        } else {
            const int px[3] = {sc.x + 1, sc.x == Lx - 1 ? 0 : -1, sc.x == 0 ? Lx + 1 : -1};
            const int py[3] = {sc.y + 1, sc.y == Ly - 1 ? 0 : -1, sc.y == 0 ? Ly + 1 : -1};
            const int pz[3] = {sc.z + 1, sc.z == Lz - 1 ? 0 : -1, sc.z == 0 ? Lz + 1 : -1};
            for (int ix = 0; ix < 3; ++ix)
                for (int iy = 0; iy < 3; ++iy)
                    for (int iz = 0; iz < 3; ++iz) {
                        if (px[ix] < 0 || py[iy] < 0 || pz[iz] < 0) continue;
                        const uint32_t pi = (uint32_t)((((px[ix] * G.PLy + py[iy]) * G.PLz + pz[iz]) << LC::lgA) | sc.b);
                        occ_set<OCC>(s_occ, pi, code);
                    }
        }
    };
    // the two sites of a move and all their neighbours are now "touched" (pipelined accept engine); lanes 0..31 of one warp
    auto mark_one = [&](uint32_t u, int lane) {
        const SiteC sc = decode_site<LAT>(G, u);
        const bool interior = sc.x >= 1 && sc.x <= Lx - 2 && sc.y >= 1 && sc.y <= Ly - 2 && sc.z >= 1 && sc.z <= Lz - 2;
        for (int e = lane; e < P.Z; e += 32) {
            const uint32_t v = interior ? u + (uint32_t)s_loff[sc.b * P.Z + e] : (uint32_t)__ldg(P.nbr_site + (size_t)u * P.Z + e);
            mark_bits(v);
        }
        if (lane == 0) mark_bits(u);
    };
    auto mark_touched = [&](uint32_t ma, uint32_t mb, int lane) {
        mark_one(ma, lane);
        mark_one(mb, lane);
    };
    // D9.4: apply an accepted move in every thread of the block (counts by the first S*M*M threads, the swap with its
    // ghost images by thread T-1, bookkeeping by thread T-2); ends with a barrier.
    auto apply_move = [&](const MoveRec* mv, uint32_t kk, unsigned long long step) {
        const int p = (int)(mv->pq & 0xFFu), q = (int)(mv->pq >> 8);
        for (int idx = tid; idx < SMM; idx += T) {
            const int s = idx / MM, rem = idx - s * MM, i = rem / M, jj = rem - i * M;
            const PW d = (PW)mv->d[s];
            const int ci = (i == p) - (i == q), cj = (jj == p) - (jj == q);
            sh.cnt[idx] += ci * Pack<M>::field(d, jj) + cj * Pack<M>::field(d, i);
        }
        if (tid == T - 1) {
            write_site(mv->a, 1u << q);
            write_site(mv->b, 1u << p);
        }
        if (AA.pae && tid >= 32 && tid < 64) mark_touched(mv->a, mv->b, tid - 32);
        if (tid == T - 2) {
            const uint32_t a = mv->a, b = mv->b;
            sh.J = mv->J;
            sh.bestk = kNoKey; sh.bestJ = ~0ull;
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
        __syncthreads();
    };

    // D9.1: the proposal of candidate (step, k): sites, their decoded positions and one-hot species (equal codes = null)
    auto propose2 = [&](unsigned long long step, uint32_t k, uint32_t& a, uint32_t& b, SiteC& sa, SiteC& sb, uint32_t& hp,
                        uint32_t& hq, uint32_t& a1, uint32_t& b1) {
        const uint4 r = philox4x32_10_rk((uint32_t)step, (uint32_t)(step >> 32), k, chain, AA.rk);
        a = __umulhi(r.x, (uint32_t)N); b = __umulhi(r.y, (uint32_t)N - 1u);
        b += (b >= a);
        a1 = a; b1 = b;
        sa = decode_site<LAT>(G, a); sb = decode_site<LAT>(G, b);
        hp = occ_get<OCC>(s_occ, sa.pidx); hq = occ_get<OCC>(s_occ, sb.pidx);
        if (hp == hq) {
            a = __umulhi(r.z, (uint32_t)N); b = __umulhi(r.w, (uint32_t)N - 1u);
            b += (b >= a);
            sa = decode_site<LAT>(G, a); sb = decode_site<LAT>(G, b);
            hp = occ_get<OCC>(s_occ, sa.pidx); hq = occ_get<OCC>(s_occ, sb.pidx);
        }
    };
    auto propose = [&](unsigned long long step, uint32_t k, uint32_t& a, uint32_t& b, SiteC& sa, SiteC& sb, uint32_t& hp,
                       uint32_t& hq) {
        uint32_t a1, b1;
        propose2(step, k, a, b, sa, sb, hp, hq, a1, b1);
    };
    // D9.2: per shell, (entries of a's row equal to b) - (entries of a row equal to its own site)
    auto adjacency = [&](uint32_t a, uint32_t b, const SiteC& sa, const SiteC& sb, int& mm0, int& mm1, int& mm2) {
        mm0 = 0; mm1 = 0; mm2 = 0;
        if (G.distinct) {
            // neighbours of any shell sit in cells at most one apart (periodically): almost every pair fails on x or y
            const int cx = sb.x - sa.x, cy = sb.y - sa.y;
            const int ax = abs(cx), ay = abs(cy);
            if ((ax <= 1 || ax == Lx - 1) && (ay <= 1 || ay == Ly - 1)) {
                const int cz = sb.z - sa.z;
                const int dx = 2 * cx + (int)((G.basis >> (3 * sb.b)) & 1u) - (int)((G.basis >> (3 * sa.b)) & 1u);
                const int dy = 2 * cy + (int)((G.basis >> (3 * sb.b + 1)) & 1u) - (int)((G.basis >> (3 * sa.b + 1)) & 1u);
                const int dz = 2 * cz + (int)((G.basis >> (3 * sb.b + 2)) & 1u) - (int)((G.basis >> (3 * sa.b + 2)) & 1u);
                const int wx = dx > Lx ? dx - 2 * Lx : dx < -Lx ? dx + 2 * Lx : dx;
                const int wy = dy > Ly ? dy - 2 * Ly : dy < -Ly ? dy + 2 * Ly : dy;
                const int wz = dz > Lz ? dz - 2 * Lz : dz < -Lz ? dz + 2 * Lz : dz;
                const int r2 = wx * wx + wy * wy + wz * wz;
                mm0 = r2 == G.d2[0]; mm1 = r2 == G.d2[1]; mm2 = r2 == G.d2[2];
            }
        } else {
            const int32_t* row = nbr + (size_t)a * P.Z;
            for (int e = 0; e < P.Z; ++e) {
                const int hit = (uint32_t)__ldg(row + e) == b;
                if (e < P.zoff[1]) mm0 += hit; else if (e < P.zoff[2]) mm1 += hit; else mm2 += hit;
            }
            mm0 -= P.m_self[0]; mm1 -= P.m_self[1]; mm2 -= P.m_self[2];
        }
    };

    // ---- site-histogram table of the reject filter.  The filter needs, per candidate, only the species
    // of the two sites and the difference of their first-shell neighbour counts.  Both are kept PER SITE in a 32-bit word
    // (species << 24 | counts of species 0..M-2) in global memory, read through L2: a candidate of a long window is then
    // Philox, two loads and the fp32 form -- no site decode, no gathers.  Moves are rare where long windows run, and a move
    // changes the words of its two sites and of their 2 z_1 neighbours, which are recomputed from the configuration.
    // Every block of a team writes the same values (its replica of the configuration is the same), so no block waits
    // for another: its own stores are fenced before its next window, and the window exchange orders the stores of
    // consecutive moves.  The table is built when a phase of long windows starts (each block a slice, then a team barrier).
    constexpr int HFB = M <= 4 ? 8 : 6;
    constexpr uint32_t HFM = (1u << HFB) - 1u;
    uint32_t* const g_hist = (M >= 2 && M <= 5 && AA.hist != nullptr && G.distinct) ? AA.hist + chain_local * (size_t)N : nullptr;
    bool hist_valid = false, hist_pending = false;
    uint32_t hist_a = 0u, hist_b = 0u, hist_epoch = 0u;
    auto hist_word = [&](uint32_t site) -> uint32_t {
        const SiteC sc = decode_site<LAT>(G, site);
        uint32_t acc[NA0];
        gather_first_direct<OCC, NA0>(s_occ, sh.fs_rd[sc.b], sc.pidx, AA.fs_c, acc);
        uint32_t h = (uint32_t)(31 - __clz((int)occ_get<OCC>(s_occ, sc.pidx))) << 24;
#pragma unroll
        for (int r = 0; r < M - 1; ++r) {
            uint32_t x = 0u;
#pragma unroll
            for (int g = 0; g < NA0; ++g) x += (acc[g] >> r) & 0x01010101u;
            h |= ((x * 0x01010101u) >> 24) << (HFB * r);
        }
        return h;
    };
    auto hist_build = [&]() {
        const uint32_t per = ((uint32_t)N + (uint32_t)R - 1u) / (uint32_t)R;
        const uint32_t lo = rank * per, hi = min((uint32_t)N, lo + per);
        for (uint32_t i = lo + (uint32_t)tid; i < hi; i += (uint32_t)T) __stcg(g_hist + i, hist_word(i));
        __threadfence();
        __syncthreads();
        if (R > 1) {
            ++hist_epoch;
            if (tid == 0) {
                __threadfence();
                atomicAdd(&ctl->hist_bar, 1u);
                while (ld_acquire_u32(&ctl->hist_bar) < hist_epoch * (uint32_t)R) { }
            }
            __syncthreads();
        }
    };
    // the words of the two sites of a move and of their first-shell neighbours, by the last warp of the block
    auto hist_update = [&](uint32_t ma, uint32_t mb) {
        if (tid >= T - 32) {
            for (int e = tid - (T - 32); e < 2 * LC::z0 + 2; e += 32) {
                const uint32_t v = e < LC::z0       ? (uint32_t)__ldg(nbr + (size_t)ma * P.Z + e)
                                 : e < 2 * LC::z0   ? (uint32_t)__ldg(nbr + (size_t)mb * P.Z + (e - LC::z0))
                                 : e == 2 * LC::z0  ? ma : mb;
                __stcg(g_hist + v, hist_word(v));
            }
            __threadfence();
        }
    };

    // ---- accept engine: one candidate per group of 8 lanes (latency instead of throughput).  Every lane of a group
    // draws the same proposal; the accumulator words of the 2Z gathers and the S*M rows of the objective are dealt
    // over the lanes; species counts are combined by xor-shuffles, the rows in the D6 order by indexed shuffles.
    using PD = typename std::conditional<(M <= 5), uint32_t, uint64_t>::type;     // (M-1) 8-bit fields
    constexpr int NWR = (2 * (NA0 + NA1 + NA2) + 7) / 8;                          // word rounds per lane
    constexpr int NRR = (3 * M + 7) / 8;                                          // row rounds per lane
    const int nw = 2 * (NA0 + (S > 1 ? NA1 : 0) + (S > 2 ? NA2 : 0));
    // species-count differences of all shells for the candidate (sa, sb), the 8 lanes of a group sharing the gathers
    auto g8_F = [&](const SiteC& sa, const SiteC& sb, int mm0, int mm1, int mm2, int p, int q, int (&c)[M], int (&F0)[M],
                    int (&F1)[M], int (&F2)[M]) {
        const int l8 = tid & 7;
        // gathers: this lane's accumulator words -> biased species counts (+ for b's neighbours, - for a's)
        PD D0 = 0, D1 = 0, D2 = 0;
        PD bias4 = 0;
#pragma unroll
        for (int r2 = 0; r2 < M - 1; ++r2) bias4 |= (PD)4 << (8 * r2);
#pragma unroll
        for (int rd = 0; rd < NWR; ++rd) {
            const int w = l8 + 8 * rd;
            if (w < nw) {
                const int4 dsc = sh.wdesc[w];
                const uint32_t pidx = dsc.w ? sb.pidx : sa.pidx;
                const int bb = dsc.w ? sb.b : sa.b;
                const int4 o = reinterpret_cast<const int4*>(s_tab + bb * ZP)[dsc.x];
                const uint8_t* base = s_occ + (OCC == OCC2_NIB ? pidx >> 1 : pidx);
                uint32_t acc = 0;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int oj = j == 0 ? o.x : j == 1 ? o.y : j == 2 ? o.z : o.w;
                    acc += (uint32_t)base[OCC == OCC2_NIB ? (oj >> 3) : oj] << (8 * j);
                }
                if (OCC == OCC2_NIB) acc = (acc >> (o.x & 4)) & 0x0F0F0F0Fu;   // a group shares its nibble shift (table order)
                acc &= (uint32_t)dsc.y;
                PD pk = 0;
#pragma unroll
                for (int r2 = 0; r2 < M - 1; ++r2)
                    pk |= (PD)((((acc >> r2) & 0x01010101u) * 0x01010101u) >> 24) << (8 * r2);
                const PD v = dsc.w ? bias4 + pk : bias4 - pk;
                D0 += dsc.z == 0 ? v : (PD)0; D1 += dsc.z == 1 ? v : (PD)0; D2 += dsc.z == 2 ? v : (PD)0;
            }
        }
#pragma unroll
        for (int o = 1; o < 8; o <<= 1) {
            D0 += __shfl_xor_sync(0xFFFFFFFFu, D0, o);
            if (S > 1) D1 += __shfl_xor_sync(0xFFFFFFFFu, D1, o);
            if (S > 2) D2 += __shfl_xor_sync(0xFFFFFFFFu, D2, o);
        }
        {
            int l0 = 0, l1 = 0, l2 = 0;
#pragma unroll
            for (int r2 = 0; r2 < M; ++r2) {
                c[r2] = (r2 == p) - (r2 == q);
                if (r2 < M - 1) {
                    F0[r2] = (int)((D0 >> (8 * r2)) & 0xFFu) - 8 * NA0; l0 -= F0[r2];
                    F1[r2] = (int)((D1 >> (8 * r2)) & 0xFFu) - 8 * NA1; l1 -= F1[r2];
                    F2[r2] = (int)((D2 >> (8 * r2)) & 0xFFu) - 8 * NA2; l2 -= F2[r2];
                } else {
                    F0[r2] = l0; F1[r2] = l1; F2[r2] = l2;
                }
            }
            if (S < 2) {
#pragma unroll
                for (int r2 = 0; r2 < M; ++r2) F1[r2] = 0;
            }
            if (S < 3) {
#pragma unroll
                for (int r2 = 0; r2 < M; ++r2) F2[r2] = 0;
            }
#pragma unroll
            for (int r2 = 0; r2 < M; ++r2) { F0[r2] -= mm0 * c[r2]; F1[r2] -= mm1 * c[r2]; F2[r2] -= mm2 * c[r2]; }
        }
    };
    // J of the candidate from the current counts and its F, rows dealt over the 8 lanes, combined in the D6 order
    auto g8_J = [&](const int (&c)[M], int p, int q, const int (&F0)[M], const int (&F1)[M], const int (&F2)[M]) -> double {
        const int l8 = tid & 7;
        // rows of the objective: row rho = s*M + i on lane rho & 7
        double rowv[NRR];
#pragma unroll
        for (int rr = 0; rr < NRR; ++rr) {
            const int rho = l8 + 8 * rr;
            double row = 0.0;
            if (rho < S * M) {
                const int s = rho / M, i = rho - s * M;
                const int ci = (i == p) - (i == q);
                int Fi = 0;
#pragma unroll
                for (int j = 0; j < M; ++j) { const int Fj = s == 0 ? F0[j] : s == 1 ? F1[j] : F2[j]; Fi = j == i ? Fj : Fi; }
#pragma unroll
                for (int j = 0; j < M; ++j) {
                    const int Fj = s == 0 ? F0[j] : s == 1 ? F1[j] : F2[j];
                    const int n = sh.cnt[rho * M + j] + ci * Fj + c[j] * Fi;
                    row = __dadd_rn(row, sq_dev(n, sh.g[rho * M + j], sh.t[rho * M + j]));
                }
            }
            rowv[rr] = row;
        }
        // D6 combination: rows in order within a shell, shells in order
        double Jk = 0.0;
#pragma unroll
        for (int s = 0; s < 3; ++s) {
            if (s < S) {
                double shs = 0.0;
#pragma unroll
                for (int i = 0; i < M; ++i) {
                    constexpr int dummy = 0; (void)dummy;
                    const int rho = s * M + i;
                    const double v = __shfl_sync(0xFFFFFFFFu, rowv[rho >> 3], (tid & 24) | (rho & 7));
                    shs = __dadd_rn(shs, v);
                }
                Jk = __dadd_rn(Jk, __dmul_rn(Kc.w[s], shs));
            }
        }
        return Jk;
    };
    auto g8_post = [&](bool live, double Jk, double J_cur, uint32_t k, uint32_t a, uint32_t b, int p, int q,
                       const int (&F0)[M], const int (&F1)[M], const int (&F2)[M], int grp, int buf) {
        const int l8 = tid & 7;
        if (l8 == 0 && live && Jk < J_cur) {
            MoveRec& m = sh.cand[grp];
            m.key = k; m.a = a; m.b = b; m.pq = (uint32_t)p | ((uint32_t)q << 8); m.J = Jk;
            m.d[0] = pack_F<M>(F0); m.d[1] = pack_F<M>(F1); m.d[2] = pack_F<M>(F2);
            atomicMin(&sh.best[buf], k);
        }
    };
    auto eval_g8 = [&](unsigned long long step, uint32_t k, bool valid, int grp, int buf, double J_cur) {
        uint32_t a, b, hp, hq;
        SiteC sa, sb;
        propose(step, k, a, b, sa, sb, hp, hq);
        const bool live = valid && hp != hq;
        const int p = 31 - __clz((int)hp), q = 31 - __clz((int)hq);
        int mm0, mm1, mm2;
        adjacency(a, b, sa, sb, mm0, mm1, mm2);
        int c[M], F0[M], F1[M], F2[M];
        g8_F(sa, sb, mm0, mm1, mm2, p, q, c, F0, F1, F2);
        const double Jk = g8_J(c, p, q, F0, F1, F2);
        g8_post(live, Jk, J_cur, k, a, b, p, q, F0, F1, F2, grp, buf);
    };

    unsigned long long t0 = A.step0;
    const unsigned long long t_end = A.step0 + A.n_steps;
    uint32_t W = 1;
    unsigned long long my_null = 0;
    uint32_t it = 0;                                         // windows evaluated by this block
    uint32_t tw = 0;                                         // TEAM windows so far (same in every block of the team)
    uint32_t phase = 0;                                      // phase records consumed / posted
    double slack_J = -1.0;                                   // J the pre-filter intervals were computed for (J >= 0 always)

    while (t0 < t_end && !(depth_limit && depth >= depth_limit)) {
        if (R > 1 && !team && rank != 0) {
            // ---- follower in a SOLO phase: wait for the leader's phase record, reload, join the team
            if (tid == 0) {
                while (ld_acquire_u32(&ctl->phase_seq) != phase + 1u) __nanosleep(256);
                sh.bc_W = __ldcg(&ctl->W);                   // broadcast through shared memory
                sh.bc_t0 = __ldcg(&ctl->t0);
                sh.bc_depth = __ldcg(&ctl->depth);
                sh.J = __ldcg(&ctl->J);
            }
            __syncthreads();
            ++phase;
            W = sh.bc_W;
            t0 = sh.bc_t0;
            depth = sh.bc_depth;
            if (t0 >= t_end) break;
            load_state();
            set_mode(true);
            __syncthreads();
            continue;
        }
        uint32_t key_best = kNoKey, steps_done = 1u;
        if (accept_ok && !team && W == 1u && AA.pae) {
            hist_valid = false; hist_pending = false;            // moves of this engine do not maintain the site histograms
            // ---- serial accept engine.  In the accept regime nearly every step applies a move found among its first few
            // candidates, so a chain advances one dependent move at a time and what counts is the latency of a step.
            // (P) What depends only on the configuration (proposal, adjacency, the 2Z gathers) is computed AHEAD for an
            //     epoch of T / 16 steps x 16 candidates by the whole block, one record per thread.
            // (S) FOUR warps (16 records x 8 lanes) then run the steps of the epoch, synchronised among themselves by a
            //     named barrier while the other warps wait: the objective of the records against the current counts, the
            //     lowest improving candidate, then counts, configuration, bitmap and bookkeeping dealt over the four
            //     warps.  A record is stale once a move has touched one of its drawn sites or one of their neighbours (a
            //     bitmap marked by every move); stale records below the first improving one are rebuilt from the
            //     current configuration.  A step whose first 16 candidates do not improve goes to the whole block
            //     (rounds of 32 candidates, 8 lanes each).
            // (N) The null candidates of the consumed steps (all K count, D9.1) are settled afterwards by the whole
            //     block against the final configuration, sites touched by moves of the epoch being traced back
            //     through the epoch's move log.
            const uint32_t n_ep = (uint32_t)min((unsigned long long)(T / kPaeK), t_end - t0);
            const unsigned long long t_ep = t0;
            auto px_of = [&](const SiteC& sc) -> uint32_t {
                const bool interior = sc.x >= 1 && sc.x <= Lx - 2 && sc.y >= 1 && sc.y <= Ly - 2 && sc.z >= 1 && sc.z <= Lz - 2;
                return sc.pidx | (interior ? 0x80000000u : 0u);
            };
            auto build_record = [&](unsigned long long step, uint32_t k, uint2& px) -> PRec {
                PRec rec;
                px = make_uint2(0u, 0u);
                rec.pad = 0; rec.d0 = rec.d1 = rec.d2 = 0ull; rec.a = rec.b = rec.a1 = rec.b1 = 0u;
                rec.pqn = 1u << 17;                                   // absent (k >= K)
                if (k < (uint32_t)K) {
                    uint32_t a, b, hp, hq, a1, b1;
                    SiteC sa, sb;
                    propose2(step, k, a, b, sa, sb, hp, hq, a1, b1);
                    rec.a = a; rec.b = b; rec.a1 = a1; rec.b1 = b1;
                    px = make_uint2(px_of(sa), px_of(sb));
                    if (hp == hq) {
                        rec.pqn = 1u << 16;                           // null
                    } else {
                        const int p = 31 - __clz((int)hp), q = 31 - __clz((int)hq);
                        int c[M], F0[M], F1[M], F2[M];
#pragma unroll
                        for (int r2 = 0; r2 < M; ++r2) { c[r2] = (r2 == p) - (r2 == q); F1[r2] = 0; F2[r2] = 0; }
                        int mm0, mm1, mm2;
                        adjacency(a, b, sa, sb, mm0, mm1, mm2);
                        const int4* ta = reinterpret_cast<const int4*>(s_tab + sa.b * ZP);
                        const int4* tb = reinterpret_cast<const int4*>(s_tab + sb.b * ZP);
                        {
                            uint32_t xa[NA0], xb[NA0];
                            gather_shell<OCC, LC::z0>(s_occ, ta, sa.pidx, xa);
                            gather_shell<OCC, LC::z0>(s_occ, tb, sb.pidx, xb);
                            hist_diff<M, NA0>(xa, xb, F0);
                        }
                        if (S > 1) {
                            uint32_t xa[NA1], xb[NA1];
                            gather_shell<OCC, LC::z1>(s_occ, ta + NA0, sa.pidx, xa);
                            gather_shell<OCC, LC::z1>(s_occ, tb + NA0, sb.pidx, xb);
                            hist_diff<M, NA1>(xa, xb, F1);
                        }
                        if (S > 2) {
                            uint32_t xa[NA2], xb[NA2];
                            gather_shell<OCC, LC::z2>(s_occ, ta + NA0 + NA1, sa.pidx, xa);
                            gather_shell<OCC, LC::z2>(s_occ, tb + NA0 + NA1, sb.pidx, xb);
                            hist_diff<M, NA2>(xa, xb, F2);
                        }
#pragma unroll
                        for (int r2 = 0; r2 < M; ++r2) { F0[r2] -= mm0 * c[r2]; F1[r2] -= mm1 * c[r2]; F2[r2] -= mm2 * c[r2]; }
                        rec.pqn = (uint32_t)p | ((uint32_t)q << 8);
                        rec.d0 = (unsigned long long)pack_F<M>(F0); rec.d1 = (unsigned long long)pack_F<M>(F1);
                        rec.d2 = (unsigned long long)pack_F<M>(F2);
                    }
                }
                return rec;
            };
            if ((uint32_t)tid < n_ep * (uint32_t)kPaeK) {
                uint2 px;
                s_prec[tid] = build_record(t0 + (uint32_t)tid / (uint32_t)kPaeK, (uint32_t)tid % (uint32_t)kPaeK, px);
                s_px[tid] = px;
            }
            if (tid < kPaeRecs / kPaeK) sh.mlog[tid] = make_uint4(0u, 0u, 0u, 0u);
            for (int i = tid; i < kDirty2Words; i += T) s_dirty2[i] = 0u;   // the queue's words: dead between windows
            mark2 = true;
            __syncthreads();
            uint32_t e_done = 0;                                         // steps of the epoch consumed
            bool leave = false;
            while (e_done < n_ep && !leave) {
                // warps 0-3 (EVAL): 16 records x 8 lanes, the pair counts of a lane's objective rows in registers.
                // warps 4-7 (ROLES): what a move changes besides the counts -- touched-site bitmap (warps 4, 5), the swap
                // with its ghost images (warp 6), shared counts, J, hash, logs (warp 7) -- one step behind the evaluation.
                // Named barriers: 2 = "bitmap and configuration of the previous move are in place" (roles arrive, eval
                // waits), 3 = "selection of this step posted" (all eight warps), 4 = the same after rebuilt records.
                // An improving group posts its J and, per objective row, the count changes as packed signed bytes
                // (s_dn); the move itself is read from the record of the winner.
                if (tid < 256) {
                    const bool is_eval = tid < 128;
                    const int grp = (tid >> 3) & 15, l8 = tid & 7;
                    const int SMr = S * M;
                    auto dirty = [&](uint32_t v) { return touched(v); };
                    auto sext8 = [](unsigned long long v, int j) { return (int)(signed char)(unsigned char)(v >> (8 * j)); };
                    int cntr[NRR][M];                                    // EVAL: counts of rows l8 + 8 rr
                    int srow[NRR], irow[NRR];
#pragma unroll
                    for (int rr = 0; rr < NRR; ++rr) {
                        const int rho = l8 + 8 * rr;
                        const bool v = is_eval && rho < SMr;
                        srow[rr] = v ? rho / M : -1;
                        irow[rr] = v ? rho - srow[rr] * M : 0;
#pragma unroll
                        for (int j = 0; j < M; ++j) cntr[rr][j] = v ? sh.cnt[rho * M + j] : 0;
                    }
                    // J and packed count changes of a candidate (pqn, packed F of the shells of this lane's rows)
                    auto eval_rows = [&](uint32_t pqn, const unsigned long long (&dsel)[NRR], unsigned long long (&dnp)[NRR]) -> double {
                        const bool live = !((pqn >> 16) & 3u);
                        const int p = (int)(pqn & 0xFFu), q = (int)((pqn >> 8) & 0xFFu);
                        double rowv[NRR];
#pragma unroll
                        for (int rr = 0; rr < NRR; ++rr) {
                            double row = 0.0;
                            unsigned long long pk = 0ull;
                            if (srow[rr] >= 0) {
                                const int i = irow[rr], rho = l8 + 8 * rr;
                                const PW d = (PW)dsel[rr];
                                const int ci = live ? (i == p) - (i == q) : 0;
                                const int Fi = (int)((d >> (Pack<M>::FB * i)) & (PW)((1 << Pack<M>::FB) - 1)) - Pack<M>::kHalf;
#pragma unroll
                                for (int j = 0; j < M; ++j) {
                                    const int cj = live ? (j == p) - (j == q) : 0;
                                    const int dn = ci * Pack<M>::field(d, j) + cj * Fi;
                                    pk |= (unsigned long long)(unsigned char)dn << (8 * j);
                                    row = __dadd_rn(row, sq_dev(cntr[rr][j] + dn, sh.g[rho * M + j], sh.t[rho * M + j]));
                                }
                            }
                            rowv[rr] = row;
                            dnp[rr] = pk;
                        }
                        double Jk = 0.0;
#pragma unroll
                        for (int s = 0; s < 3; ++s) {
                            if (s < S) {
                                double shs = 0.0;
#pragma unroll
                                for (int i = 0; i < M; ++i) {
                                    const int rho = s * M + i;
                                    const double v = __shfl_sync(0xFFFFFFFFu, rowv[rho >> 3], (tid & 24) | (rho & 7));
                                    shs = __dadd_rn(shs, v);
                                }
                                Jk = __dadd_rn(Jk, __dmul_rn(Kc.w[s], shs));
                            }
                        }
                        return Jk;
                    };
                    double J_cur = sh.J;
                    if (tid < 3) { sh.sel[tid] = make_uint2(kNoKey, 0u); sh.sbest2[tid] = kNoKey; }
                    asm volatile("bar.sync 4, 256;" ::: "memory");
                    if (!is_eval && tid < 224) asm volatile("bar.arrive 2, 224;" ::: "memory");
                    uint32_t es = e_done, pend = 0u, sit = 0u;
                    for (; es < n_ep; ++es, ++sit) {
                        const int sb = (int)(sit % 3u), par = (int)(sit & 1u);
                        const unsigned long long step = t_ep + es;
                        PRec* const rp = &s_prec[es * kPaeK + grp];
                        unsigned long long dnp[NRR];
                        double Jk = 0.0;
                        if (is_eval) {
                            const uint4 sites = *reinterpret_cast<const uint4*>(rp);     // a, b, a1, b1
                            const uint32_t pqn = rp->pqn;
                            unsigned long long dsel[NRR];
#pragma unroll
                            for (int rr = 0; rr < NRR; ++rr) dsel[rr] = (&rp->d0)[max(srow[rr], 0)];
                            Jk = eval_rows(pqn, dsel, dnp);
                            asm volatile("bar.sync 2, 224;" ::: "memory");       // the previous move is in the bitmap
                            const bool absent = (pqn >> 17) & 1u;
                            const bool stale = !absent && (dirty(sites.x) | dirty(sites.y) | dirty(sites.z) | dirty(sites.w));
                            if (stale) {
                                if (l8 == 0) atomicOr(&sh.sel[sb].y, 1u << grp);
                            } else if (!((pqn >> 16) & 3u) && Jk < J_cur) {
#pragma unroll
                                for (int rr = 0; rr < NRR; ++rr)
                                    if (srow[rr] >= 0) s_dn[(par * kPaeK + grp) * SMr + l8 + 8 * rr] = dnp[rr];
                                if (l8 == 0) { sh.sJ[par][grp] = Jk; atomicMin(&sh.sel[sb].x, (uint32_t)grp); }
                            }
                        }
                        asm volatile("bar.sync 3, 256;" ::: "memory");           // selection posted
                        const uint2 sel = sh.sel[sb];
                        uint32_t kb = sel.x;
                        // stale records below the first improving fresh one decide the step: their warps rebuild their
                        // four records from the current configuration (8 lanes per record) and evaluate again
                        const uint32_t need = sel.y & (kb == kNoKey ? 0xFFFFFFFFu : ((1u << kb) - 1u));
                        if (need) {
                            if (is_eval && ((need >> (grp & ~3)) & 0xFu)) {
                                uint32_t a, b, hp, hq;
                                SiteC sa, sb2;
                                propose(step, (uint32_t)grp, a, b, sa, sb2, hp, hq);
                                const bool absent = (rp->pqn >> 17) & 1u;
                                const bool live = !absent && hp != hq;
                                const int p = 31 - __clz((int)hp), q = 31 - __clz((int)hq);
                                int c[M], F0[M], F1[M], F2[M];
                                int mm0, mm1, mm2;
                                adjacency(a, b, sa, sb2, mm0, mm1, mm2);
                                g8_F(sa, sb2, mm0, mm1, mm2, p, q, c, F0, F1, F2);
                                const unsigned long long d0 = pack_F<M>(F0), d1 = pack_F<M>(F1), d2 = pack_F<M>(F2);
                                const uint32_t pqn = absent ? (1u << 17) : !live ? (1u << 16) : ((uint32_t)p | ((uint32_t)q << 8));
                                unsigned long long dsel[NRR];
#pragma unroll
                                for (int rr = 0; rr < NRR; ++rr) dsel[rr] = srow[rr] == 1 ? d1 : srow[rr] == 2 ? d2 : d0;
                                Jk = eval_rows(pqn, dsel, dnp);
                                if (l8 == 0) {
                                    rp->a = a; rp->b = b; rp->pqn = pqn; rp->d0 = d0; rp->d1 = d1; rp->d2 = d2;
                                    s_px[es * kPaeK + grp] = make_uint2(px_of(sa), px_of(sb2));
                                }
                                if (live && Jk < J_cur) {
#pragma unroll
                                    for (int rr = 0; rr < NRR; ++rr)
                                        if (srow[rr] >= 0) s_dn[(par * kPaeK + grp) * SMr + l8 + 8 * rr] = dnp[rr];
                                    // (a slot of its own: the readers of barrier 3 still compare sel)
                                    if (l8 == 0) { sh.sJ[par][grp] = Jk; atomicMin(&sh.sbest2[sb], (uint32_t)grp); }
                                }
                            }
                            asm volatile("bar.sync 4, 256;" ::: "memory");
                            kb = min(kb, sh.sbest2[sb]);
                        }
                        if (tid == 255) { sh.sel[(sb + 2) % 3] = make_uint2(kNoKey, 0u); sh.sbest2[(sb + 2) % 3] = kNoKey; }
                        if (kb == kNoKey) { pend = 1u; break; }
                        if (is_eval) {
                            // D9.4 on the register copy of this lane's rows
                            J_cur = sh.sJ[par][kb];
#pragma unroll
                            for (int rr = 0; rr < NRR; ++rr) {
                                if (srow[rr] >= 0) {
                                    const unsigned long long d8 = s_dn[(par * kPaeK + (int)kb) * SMr + l8 + 8 * rr];
#pragma unroll
                                    for (int j = 0; j < M; ++j) cntr[rr][j] += sext8(d8, j);
                                }
                            }
                        } else {
                            const PRec* wr = &s_prec[es * kPaeK + kb];
                            const uint32_t wa = wr->a, wb = wr->b, wpq = wr->pqn;
                            const uint2 wpx = s_px[es * kPaeK + kb];
                            const int wp = (int)(wpq & 0xFFu), wq = (int)((wpq >> 8) & 0xFFu);
                            if (tid < 192) {                             // warps 4, 5: neighbourhoods of a and of b
                                const uint32_t u = tid < 160 ? wa : wb, upx = tid < 160 ? wpx.x : wpx.y;
                                if (upx >> 31) {                         // interior cell: neighbour = site + offset of its basis index
                                    const int lane = tid & 31, bb = (int)(upx & (uint32_t)(LC::A - 1));
                                    for (int e = lane; e < P.Z; e += 32) {
                                        const uint32_t v = u + (uint32_t)s_loff[bb * P.Z + e];
                                        mark_bits(v);
                                    }
                                    if (lane == 0) mark_bits(u);
                                } else {
                                    mark_one(u, tid & 31);
                                }
                                asm volatile("bar.arrive 2, 224;" ::: "memory");
                            } else if (tid < 224) {                      // warp 6: the swap (one lane: a and b may share a byte)
                                const bool same_byte = OCC == OCC2_NIB && ((wpx.x & 0x7FFFFFFFu) >> 1) == ((wpx.y & 0x7FFFFFFFu) >> 1);
                                if ((wpx.x & wpx.y) >> 31 && !same_byte) {       // both interior: one lane each
                                    if (tid == 192) occ_set<OCC>(s_occ, wpx.x & 0x7FFFFFFFu, 1u << wq);
                                    if (tid == 193) occ_set<OCC>(s_occ, wpx.y & 0x7FFFFFFFu, 1u << wp);
                                } else if (tid == 192) {
                                    write_site(wa, 1u << wq); write_site(wb, 1u << wp);
                                }
                                asm volatile("bar.arrive 2, 224;" ::: "memory");
                            } else {                                     // warp 7: shared counts and bookkeeping
                                for (int idx = tid - 224; idx < SMM; idx += 32) {
                                    const int s2 = idx / MM, rem = idx - s2 * MM, i = rem / M, jj = rem - i * M;
                                    const PW d = (PW)(&wr->d0)[s2];
                                    const int ci = (i == wp) - (i == wq), cj = (jj == wp) - (jj == wq);
                                    sh.cnt[idx] += ci * Pack<M>::field(d, jj) + cj * Pack<M>::field(d, i);
                                }
                                if (tid == 224) {
                                    sh.J = sh.sJ[par][kb];
                                    sh.n_accept += 1;
                                    sh.last_accept = step;
                                    unsigned long long hsh = sh.hash;
                                    hsh = (hsh ^ (uint32_t)step) * 0x100000001b3ULL;
                                    hsh = (hsh ^ (uint32_t)(step >> 32)) * 0x100000001b3ULL;
                                    hsh = (hsh ^ kb) * 0x100000001b3ULL;
                                    hsh = (hsh ^ wa) * 0x100000001b3ULL;
                                    hsh = (hsh ^ wb) * 0x100000001b3ULL;
                                    sh.hash = hsh;
                                    sh.mlog[es] = make_uint4(wa, wb, (wpq & 0xFFFFu) | (1u << 16), 0u);
                                    const unsigned long long nl = sh.n_logged;
                                    if (rank == 0 && A.log_all != nullptr && (long long)nl < A.log_cap) {
                                        unsigned long long* lr = A.log_all + (chain_local * (size_t)A.log_cap + nl) * 3;
                                        lr[0] = step;
                                        lr[1] = (unsigned long long)kb | ((unsigned long long)wa << 32);
                                        lr[2] = (unsigned long long)wb;
                                    }
                                    sh.n_logged = nl + 1;
                                }
                            }
                        }
                    }
                    // barrier 2 is left balanced: one arrival is outstanding unless the loop stopped at a step without a move
                    if (is_eval && !pend) asm volatile("bar.sync 2, 224;" ::: "memory");
                    if (tid == 0) sh.swe_stop = es | (pend << 31);
                }
                __syncthreads();
                const uint32_t st = sh.swe_stop;
                if ((st & 0x7FFFFFFFu) > e_done) depth = 0;              // every step the serial engine consumed applied a move
                e_done = st & 0x7FFFFFFFu;
                if (st >> 31) {
                    // step t_ep + e_done: none of the first kPaeK candidates improves -> the others, rounds of 32 on 8 warps
                    const unsigned long long tstep = t_ep + e_done;
                    const double J_cur = sh.J;
                    uint32_t rd0 = (uint32_t)kPaeK;
                    key_best = kNoKey;
                    for (; rd0 < (uint32_t)K; rd0 += 32u) {
                        const int buf = (int)(it % 3u);
                        if (tid < 256) {
                            const uint32_t k = rd0 + ((uint32_t)tid >> 3);
                            eval_g8(tstep, k, k < (uint32_t)K, tid >> 3, buf, J_cur);
                        }
                        __syncthreads();
                        key_best = sh.best[buf];
                        if (tid == 0) { sh.best[(buf + 2) % 3] = kNoKey; sh.q_n[(buf + 2) % 3] = 0u; }
                        ++it;
                        if (key_best != kNoKey) break;
                    }
                    if (key_best != kNoKey) {
                        const MoveRec* mv = &sh.cand[key_best - rd0];
                        if (tid == 0) sh.mlog[e_done] = make_uint4(mv->a, mv->b, mv->pq | (1u << 16), 0u);
                        apply_move(mv, key_best, tstep);                 // ends with a barrier
                        depth = 0;
                    } else {
                        W = min(2u, w_cap);
                        depth += 1;
                        leave = true;
                    }
                    e_done += 1;
                }
            }
            // ---- (N) null candidates of the e_done consumed steps, all K of each.  The species of a drawn site at its
            // step is the final one unless a move of the epoch touched the site (the bitmap says so, conservatively):
            // then the moves from the end of the epoch back to that step are undone for this site.
            {
                static_assert(kPaeRecs / kPaeK == 32, "the epoch's move log is scanned one entry per lane");
                const uint32_t n_cand = e_done * (uint32_t)K;
                const int lane = tid & 31;
                const uint4 my_log = sh.mlog[lane];
                const bool my_log_valid = ((my_log.z >> 16) & 1u) && (uint32_t)lane < e_done;
                // species code of `site` as step e_at saw it; every lane of the warp takes part
                auto species_at = [&](uint32_t site, uint32_t e_at) -> uint32_t {
                    uint32_t code = occ_get<OCC>(s_occ, decode_site<LAT>(G, site).pidx);
                    uint32_t todo = __ballot_sync(0xFFFFFFFFu, touched(site) != 0u);
                    while (todo) {                                   // flagged lanes, one at a time: 32 lanes x 32 log entries
                        const int src = __ffs((int)todo) - 1;
                        todo &= todo - 1u;
                        const uint32_t s_site = __shfl_sync(0xFFFFFFFFu, site, src), s_e = __shfl_sync(0xFFFFFFFFu, e_at, src);
                        const bool in_range = my_log_valid && (uint32_t)lane >= s_e;
                        const uint32_t hit_a = __ballot_sync(0xFFFFFFFFu, in_range && my_log.x == s_site);
                        const uint32_t hit_b = __ballot_sync(0xFFFFFFFFu, in_range && my_log.y == s_site);
                        if (hit_a | hit_b) {
                            // the earliest move at or after e_at that touches the site: before it, a held p and b held q
                            const int e2 = __ffs((int)(hit_a | hit_b)) - 1;
                            const uint32_t pq2 = __shfl_sync(0xFFFFFFFFu, my_log.z, e2);
                            const uint32_t c2 = ((hit_a >> e2) & 1u) ? 1u << (pq2 & 0xFFu) : 1u << ((pq2 >> 8) & 0xFFu);
                            if (lane == src) code = c2;
                        }
                    }
                    return code;
                };
                // two candidates per thread and pass: two independent Philox chains and eight site look-ups in flight
                const uint32_t n_iter = (n_cand + 2u * (uint32_t)T - 1u) / (2u * (uint32_t)T);
                for (uint32_t i2 = 0; i2 < n_iter; ++i2) {
                    bool valid[2];
                    uint32_t e_at[2], sa1[2], sb1[2], sa2[2], sb2[2];
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const uint32_t cnd0 = (2u * i2 + (uint32_t)u) * (uint32_t)T + (uint32_t)tid;
                        valid[u] = cnd0 < n_cand;
                        const uint32_t cnd = valid[u] ? cnd0 : 0u;
                        e_at[u] = K == 1 ? cnd : __umulhi(cnd, AA.k_mq) >> AA.k_sq;
                        const uint32_t k = cnd - e_at[u] * (uint32_t)K;
                        const unsigned long long step = t_ep + e_at[u];
                        const uint4 r = philox4x32_10_rk((uint32_t)step, (uint32_t)(step >> 32), k, chain, AA.rk);
                        sa1[u] = __umulhi(r.x, (uint32_t)N); sb1[u] = __umulhi(r.y, (uint32_t)N - 1u);
                        sb1[u] += (sb1[u] >= sa1[u]);
                        sa2[u] = __umulhi(r.z, (uint32_t)N); sb2[u] = __umulhi(r.w, (uint32_t)N - 1u);
                        sb2[u] += (sb2[u] >= sa2[u]);
                    }
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const uint32_t h1 = species_at(sa1[u], e_at[u]), h2 = species_at(sb1[u], e_at[u]);
                        const uint32_t h3 = species_at(sa2[u], e_at[u]), h4 = species_at(sb2[u], e_at[u]);
                        my_null += (valid[u] && h1 == h2 && h3 == h4) ? 1u : 0u;
                    }
                }
            }
            __syncthreads();
            if (e_done > 0u) {                                           // new epoch, clean bitmap
                for (int i = tid; i < dwords; i += T) s_dirty[i] = 0u;
            }
            mark2 = false;
            __syncthreads();
            t0 = t_ep + e_done;
            steps_done = 0u;                                             // t0 already advanced
            key_best = kNoKey;
        } else if (accept_ok && !team && W == 1u) {
            hist_valid = false; hist_pending = false;
            // ---- accept engine: this one step, 32 candidates per round on the first 8 warps; the other warps settle
            // which candidates of the step are null (all K count, D9.1)
            const double J_cur = sh.J;
            if (tid >= 256) {
                for (uint32_t k = (uint32_t)tid - 256u; k < (uint32_t)K; k += (uint32_t)T - 256u) {
                    const uint4 r = philox4x32_10_rk((uint32_t)t0, (uint32_t)(t0 >> 32), k, chain, AA.rk);
                    uint32_t a = __umulhi(r.x, (uint32_t)N), b = __umulhi(r.y, (uint32_t)N - 1u);
                    b += (b >= a);
                    uint32_t hp = occ_get<OCC>(s_occ, decode_site<LAT>(G, a).pidx), hq = occ_get<OCC>(s_occ, decode_site<LAT>(G, b).pidx);
                    if (hp == hq) {
                        a = __umulhi(r.z, (uint32_t)N); b = __umulhi(r.w, (uint32_t)N - 1u);
                        b += (b >= a);
                        hp = occ_get<OCC>(s_occ, decode_site<LAT>(G, a).pidx); hq = occ_get<OCC>(s_occ, decode_site<LAT>(G, b).pidx);
                    }
                    my_null += hp == hq;
                }
            }
            uint32_t rd0 = 0;
            for (; rd0 < (uint32_t)K; rd0 += 32u) {
                const int buf = (int)(it % 3u);
                if (tid < 256) {
                    const uint32_t k = rd0 + ((uint32_t)tid >> 3);
                    eval_g8(t0, k, k < (uint32_t)K, tid >> 3, buf, J_cur);
                }
                __syncthreads();
                key_best = sh.best[buf];
                if (tid == 0) { sh.best[(buf + 2) % 3] = kNoKey; sh.q_n[(buf + 2) % 3] = 0u; }
                ++it;
                if (key_best != kNoKey) break;
            }
            if (key_best != kNoKey) {
                apply_move(&sh.cand[key_best - rd0], key_best, t0);
                W = 1u;
                depth = 0;
            } else {
                W = min(2u, w_cap);
                depth += 1;
            }
        } else {
            const uint32_t Wc = (uint32_t)min(min((unsigned long long)W, t_end - t0), depth_limit ? depth_limit - depth : ~0ull);
            const int buf = (int)(it % 3u);
            volatile uint32_t* best_slot = &sh.best[buf];
            const double J_cur = sh.J;
            uint32_t win_key = kNoKey, win_a = 0, win_b = 0, win_pq = 0;
            PW win_d0 = 0, win_d1 = 0, win_d2 = 0;
            double win_J = 0.0;
            uint32_t nullw[kNullWords];                             // bit j = this thread's j-th candidate of the window is null
#pragma unroll
            for (int wd = 0; wd < kNullWords; ++wd) nullw[wd] = 0u;

            // ---- long windows run in two stages.  Stage 1: a reduced-precision REJECT FILTER on the first shell.  With
            // w_s >= 0 the first-shell term w_1 sh_1 of a candidate is a lower bound of its J_k (partial sums of D6 are
            // monotone), and in exact arithmetic it is a quadratic form of the first-shell count differences F:
            //   w_1 sh_1' = C + sum_r (L_r + Q_r F_r) F_r + X (F_q - F_p)^2,   coefficients per ordered species pair (p, q)
            // (DESIGN.md 6.2).  The form is evaluated in fp32 from a per-pair table row rebuilt after every move; the row's
            // threshold = max(1.001 J_cur, floor) - C + E rounded up (floor = 1e-18 w_1, scaled up for dilute species), where E bounds (rigorously: coefficient
            // rounding, the fp32 evaluation, the fp64 table arithmetic) the distance between the fp32 value and the exact
            // one for every admissible F, and the 0.1 % margin and the floor cover the rounding of the D6 evaluation itself.
            // A candidate above its threshold cannot improve and is dropped; the survivors are queued and evaluated exactly
            // (stage 2), so every accept decision is the fp64 one.  Needs a bit-symmetric target and w >= 0, w_1 > 0.
            const bool use_filter = SYM && prune && Kc.w[0] > 0.0 && (unsigned long long)Wc * (unsigned)K >= 2ull * GT;
            // site histograms: the filter of this window reads them when the whole team is here (a leader
            // running long windows alone must not wait for followers that wait for it)
            const bool use_hist = use_filter && g_hist != nullptr && (R == 1 || team);
            bool need_sync = false;
            if (hist_pending) { hist_update(hist_a, hist_b); hist_pending = false; need_sync = true; }
            if (use_hist && !hist_valid) { hist_build(); hist_valid = true; }
            if (use_filter && !(slack_J == J_cur)) {
                need_sync = true;
                for (int idx = tid; idx < MM; idx += T) {
                    const int p = idx / M, q = idx - p * M;
                    float* row = s_ftab + idx;                           // element e at row[e * MM]
                    double Cq = 0.0, EC = 0.0;                          // C and the bound of its own error
                    for (int c2 = 0; c2 < MM; ++c2) {
                        const double be = (double)sh.cnt[c2] - sh.nstar[c2];
                        const double eb = 4.44e-16 * (fabs(sh.nstar[c2]) + fabs(be));       // 2^-51: |be - beta| <= eb
                        Cq += sh.W1[c2] * be * be;
                        EC += sh.W1[c2] * (2.0 * fabs(be) + eb) * eb;
                    }
                    auto Wc2 = [&](int i, int j2) { return sh.W1[i * M + j2]; };
                    auto b2 = [&](int i, int j2) { return 2.0 * ((double)sh.cnt[i * M + j2] - sh.nstar[i * M + j2]); };
                    auto e2 = [&](int i, int j2) {                     // bound of the error of b2
                        return 2.0 * 4.44e-16 * (fabs(sh.nstar[i * M + j2]) + fabs((double)sh.cnt[i * M + j2] - sh.nstar[i * M + j2]));
                    };
                    const double Fm = 2.0 * (double)LC::z0;            // |F_r| <= z_1 + multiplicity corrections <= 2 z_1
                    double A = 0.0, B = 0.0;                           // sum of |term| bounds; propagated input error
                    bool finite = p != q;
                    for (int r = 0; r < M; ++r) {
                        double t1, t2, Qr, cr = 0.0, et;
                        if (r == p)      { t1 =  2.0 * Wc2(p, p) * b2(p, p); t2 = -2.0 * Wc2(p, q) * b2(p, q); Qr = 4.0 * Wc2(p, p); cr = -1.0;
                                           et = 2.0 * Wc2(p, p) * e2(p, p) + 2.0 * Wc2(p, q) * e2(p, q); }
                        else if (r == q) { t1 = -2.0 * Wc2(q, q) * b2(q, q); t2 =  2.0 * Wc2(p, q) * b2(p, q); Qr = 4.0 * Wc2(q, q); cr = 1.0;
                                           et = 2.0 * Wc2(q, q) * e2(q, q) + 2.0 * Wc2(p, q) * e2(p, q); }
                        else             { t1 =  2.0 * Wc2(p, r) * b2(p, r); t2 = -2.0 * Wc2(q, r) * b2(q, r); Qr = 2.0 * (Wc2(p, r) + Wc2(q, r));
                                           et = 2.0 * Wc2(p, r) * e2(p, r) + 2.0 * Wc2(q, r) * e2(q, r); }
                        const float Lf = (float)(t1 + t2), Qf = (float)Qr;
                        row[(2 + r) * MM] = Lf; row[(2 + M + r) * MM] = Qf; row[(2 + 2 * M + r) * MM] = (float)cr;
                        A += (fabs(t1) + fabs(t2)) * Fm + Qr * Fm * Fm;
                        B += et * Fm;
                        // a coefficient lost to fp32 underflow or overflow would break the relative-error model
                        finite = finite && isfinite(Lf) && isfinite(Qf) && (Qf >= 1.0e-30f) && (Lf == 0.0f || fabsf(Lf) >= 1.0e-30f);
                    }
                    const double X = 2.0 * Wc2(p, q);
                    const float Xf = (float)X;
                    A += X * 4.0 * Fm * Fm;
                    finite = finite && isfinite(Xf) && Xf >= 1.0e-30f;
                    // E: 2^-19 A covers the fp32 coefficient roundings and the <= 16 roundings of the fp32 evaluation
                    // (gamma_16 < 2^-20) and the fp64 roundings of the table arithmetic; B and EC the cancellation in cnt - n*
                    const double E = 1.9073486328125e-6 * A + 1.000001 * (B + EC) + 1.0e-12 * fabs(Cq);
                    const double thr = fmax(1.001 * J_cur, AA.filt_floor) - Cq + E;
                    const float thr_f = __double2float_ru(thr);
                    row[0] = (finite && isfinite(thr_f)) ? thr_f : __int_as_float(0x7f800000);   // +inf: nothing is dropped
                    row[MM] = Xf;
                }
                slack_J = J_cur;
            }
            if (need_sync) __syncthreads();
            // the part of an evaluation after the first shell's F: D6 objective shell by shell with the exact pruning
            auto eval_rest = [&](uint32_t key, uint32_t a, uint32_t b, const SiteC& sa, const SiteC& sb, int p, int q,
                                 int mm1, int mm2, const int (&F0)[M]) {
                const int4* ta = reinterpret_cast<const int4*>(s_tab + sa.b * ZP);
                const int4* tb = reinterpret_cast<const int4*>(s_tab + sb.b * ZP);
                int c[M], F1[M], F2[M];
#pragma unroll
                for (int r2 = 0; r2 < M; ++r2) { c[r2] = (r2 == p) - (r2 == q); F1[r2] = 0; F2[r2] = 0; }
                double Jk = __dmul_rn(Kc.w[0], shell_sum_F<M, SYM>(sh.cnt, Kc.g, Kc.t, F0, c));
                Jk = __dadd_rn(0.0, Jk);
                if (S > 1 && (!prune || __any_sync(__activemask(), Jk < J_cur))) {
                    {
                        uint32_t xa[NA1], xb[NA1];
                        gather_shell<OCC, LC::z1>(s_occ, ta + NA0, sa.pidx, xa);
                        gather_shell<OCC, LC::z1>(s_occ, tb + NA0, sb.pidx, xb);
                        hist_diff<M, NA1>(xa, xb, F1);
#pragma unroll
                        for (int r2 = 0; r2 < M; ++r2) F1[r2] -= mm1 * c[r2];
                    }
                    Jk = __dadd_rn(Jk, __dmul_rn(Kc.w[1], shell_sum_F<M, SYM>(sh.cnt + MM, Kc.g + MM, Kc.t + MM, F1, c)));
                    if (S > 2 && (!prune || __any_sync(__activemask(), Jk < J_cur))) {
                        {
                            uint32_t xa[NA2], xb[NA2];
                            gather_shell<OCC, LC::z2>(s_occ, ta + NA0 + NA1, sa.pidx, xa);
                            gather_shell<OCC, LC::z2>(s_occ, tb + NA0 + NA1, sb.pidx, xb);
                            hist_diff<M, NA2>(xa, xb, F2);
#pragma unroll
                            for (int r2 = 0; r2 < M; ++r2) F2[r2] -= mm2 * c[r2];
                        }
                        Jk = __dadd_rn(Jk, __dmul_rn(Kc.w[2], shell_sum_F<M, SYM>(sh.cnt + 2 * MM, Kc.g + 2 * MM, Kc.t + 2 * MM, F2, c)));
                    } else if (S > 2) {
                        Jk = J_cur;                       // pruned: not improving
                    }
                } else if (S > 1) {
                    Jk = J_cur;
                }
                // this thread keeps its best candidate: the lowest key, or in best-of-K mode the lowest (step, J, k)
                const uint32_t kts = key >> 10, wts = win_key >> 10;
                const bool better = best_mode ? (kts < wts || (kts == wts && (Jk < win_J || (Jk == win_J && key < win_key))))
                                              : key < win_key;
                if (Jk < J_cur && better) {
                    win_key = key; win_a = a; win_b = b; win_pq = (uint32_t)p | ((uint32_t)q << 8);
                    win_d0 = pack_F<M>(F0); win_d1 = pack_F<M>(F1); win_d2 = pack_F<M>(F2); win_J = Jk;
                    atomicMin(&sh.best[buf], best_mode ? (key & ~1023u) : key);
                }
            };
            // first-shell species-count differences of a non-null candidate
            auto first_shell = [&](const SiteC& sa, const SiteC& sb, int mm0, int p, int q, int (&F0)[M]) {
                uint32_t xa[NA0], xb[NA0];
                gather_first_direct<OCC, NA0>(s_occ, sh.fs_rd[sa.b], sa.pidx, AA.fs_c, xa);
                gather_first_direct<OCC, NA0>(s_occ, sh.fs_rd[sb.b], sb.pidx, AA.fs_c, xb);
                hist_diff<M, NA0>(xa, xb, F0);
                if (mm0 != 0) {                                     // a and b are first-shell neighbours (rare): D9.2 exclusion
#pragma unroll
                    for (int r2 = 0; r2 < M; ++r2) F0[r2] -= mm0 * ((r2 == p) - (r2 == q));
                }
            };

            // a queued (or overflowing) candidate, evaluated exactly from the configuration
            auto eval_key = [&](uint32_t key) {
                uint32_t a, b, hp, hq;
                SiteC sa, sb;
                propose(t0 + (key >> 10), key & 1023u, a, b, sa, sb, hp, hq);
                const int p = 31 - __clz((int)hp), q = 31 - __clz((int)hq);
                int F0[M];
                int mm0, mm1, mm2;
                adjacency(a, b, sa, sb, mm0, mm1, mm2);
                first_shell(sa, sb, mm0, p, q, F0);
                eval_rest(key, a, b, sa, sb, p, q, mm1, mm2, F0);
            };

            uint32_t ts = ts_first, k = k_first;
            uint32_t ncur = 0u;                                     // null bits of the current group of 32 candidates
            int j = 0;
            if (use_hist) {
                // ---- stage 1 from the site-histogram table: hist_scan (its own register allocation) runs this thread's
                // candidates; what it cannot settle itself (queue overflow) comes back to be evaluated here
                HistScan hs;
                hs.ts = ts_first; hs.k = k_first; hs.ncur = 0u; hs.j = 0; hs.n_ovf = 0; hs.done = 0;
#pragma unroll
                for (int wd = 0; wd < kNullWords; ++wd) hs.nullw[wd] = 0u;
                HistArgs ha;
                ha.H = g_hist; ha.rk = AA.rk; ha.best_slot = smem_addr(&sh.best[buf]); ha.ftab = smem_addr(s_ftab); ha.queue = smem_addr(sh.queue); ha.q_n = smem_addr(&sh.q_n[buf]);
                ha.t0 = t0; ha.Wc = Wc; ha.ts_inc = ts_inc; ha.k_inc = k_inc; ha.K = (uint32_t)K; ha.N = (uint32_t)N; ha.chain = chain;
                ha.Lx = Lx; ha.Ly = Ly; ha.Lz = Lz; ha.mx = G.mx; ha.sx = G.sx; ha.mq = G.mq; ha.sq = G.sq; ha.cx = G.cx; ha.cc = G.cc; ha.occ = smem_addr(s_occ); ha.basis = G.basis; ha.d2_0 = G.d2[0];
                do {
                    hist_scan<M, LAT, BEST, OCC>(hs, ha);
                    for (int i = 0; i < hs.n_ovf; ++i) eval_key(hs.ovf[i]);
                } while (!hs.done);
                j = hs.j; ncur = hs.ncur;
#pragma unroll
                for (int wd = 0; wd < kNullWords; ++wd) nullw[wd] = hs.nullw[wd];
            } else
            for (; ts < Wc; ++j) {
                const uint32_t hint = *best_slot;
                if ((hint >> 10) < ts) break;                       // a move at an earlier step exists: this step is void
                const uint32_t key = (ts << 10) | k;
                uint32_t a, b, hp, hq;
                SiteC sa, sb;
                propose(t0 + ts, k, a, b, sa, sb, hp, hq);
                ncur = __funnelshift_r(ncur, hp == hq ? 1u : 0u, 1);        // candidate j ends up at bit j & 31
                if ((j & 31) == 31) {                               // j is the same in every thread of the block
#pragma unroll
                    for (int wd = 0; wd < kNullWords; ++wd) nullw[wd] = (j >> 5) == wd ? ncur : nullw[wd];
                }
                if (hp != hq && (best_mode || key < hint)) {        // same step, higher k than a known move: only nullness counts
                    const int p = 31 - __clz((int)hp), q = 31 - __clz((int)hq);
                    int F0[M];
                    int mm0, mm1, mm2;
                    adjacency(a, b, sa, sb, mm0, mm1, mm2);
                    first_shell(sa, sb, mm0, p, q, F0);
                    bool full = true;
                    if (use_filter) {
                        const float* row = s_ftab + (p * M + q);
                        float acc = 0.0f, D = 0.0f;
#pragma unroll
                        for (int r2 = 0; r2 < M; ++r2) {
                            const float f = (float)F0[r2];
                            acc = fmaf(fmaf(row[(2 + M + r2) * MM], f, row[(2 + r2) * MM]), f, acc);
                            D = fmaf(row[(2 + 2 * M + r2) * MM], f, D);
                        }
                        acc = fmaf(row[MM] * D, D, acc);
                        full = !(acc > row[0]);
                        if (full) {
                            const uint32_t slot = atomicAdd(&sh.q_n[buf], 1u);
                            if (slot < (uint32_t)kQueueCap) { sh.queue[slot] = key; full = false; }
                        }
                    }
                    if (full) eval_rest(key, a, b, sa, sb, p, q, mm1, mm2, F0);
                }
                k += k_inc; ts += ts_inc;
                if (k >= (uint32_t)K) { k -= (uint32_t)K; ++ts; }
            }
            if (j & 31) {                                           // the last, partial group
#pragma unroll
                for (int wd = 0; wd < kNullWords; ++wd) nullw[wd] = (j >> 5) == wd ? ncur >> (32 - (j & 31)) : nullw[wd];
            }
            if (use_filter) {
                // ---- second stage: the queued survivors, one per thread
                __syncthreads();
                const uint32_t nq = min(sh.q_n[buf], (uint32_t)kQueueCap);
                for (uint32_t i = (uint32_t)tid; i < nq; i += (uint32_t)T) {
                    const uint32_t key = sh.queue[i];
                    const uint32_t hint = *best_slot;
                    if (best_mode ? (hint >> 10) < (key >> 10) : !(key < hint)) continue;
                    eval_key(key);
                }
            }
            __syncthreads();                                        // B1: window evaluated, local minimum posted
            key_best = sh.best[buf];
            if (tid == 0) { sh.best[(buf + 2) % 3] = kNoKey; sh.q_n[(buf + 2) % 3] = 0u; }   // next user of these slots is two barriers away
            if (best_mode && key_best != kNoKey) {
                // best-of-K: among this block's improving candidates of the deciding step, the minimum J, then the
                // lowest k (bestJ / bestk are reset by apply_move, which always follows)
                const bool mine = win_key != kNoKey && (win_key >> 10) == (key_best >> 10);
                if (mine) atomicMin(&sh.bestJ, ordered_bits(win_J));
                __syncthreads();
                if (mine && ordered_bits(win_J) == sh.bestJ) atomicMin(&sh.bestk, win_key);
                __syncthreads();
                key_best = sh.bestk;
            }

            const int lane = tid & 31;
            if (team) {
                // ---- TEAM exchange: post this block's best record, read all R slots, take the minimum key
                const int par = (int)(tw & 1u);
                TeamSlot* slots = ctl->slot[par];
                const bool owner = key_best != kNoKey && win_key == key_best;
                if (owner || (key_best == kNoKey && tid == 0)) {
                    TeamSlot* me = slots + rank;
                    me->key = key_best; me->a = win_a; me->b = win_b; me->pq = win_pq; me->J = win_J;
                    me->d[0] = win_d0; me->d[1] = win_d1; me->d[2] = win_d2;
                    __threadfence();
                    st_release_u32(&me->seq, tw + 1u);
                }
                if (tid < 32) {
                    uint32_t kk = kNoKey;
                    unsigned long long jb = 0ull;
                    if (lane < R) {
                        while (ld_acquire_u32(&slots[lane].seq) != tw + 1u) { }
                        kk = __ldcg(&slots[lane].key);
                        if (best_mode) jb = ordered_bits(__ldcg(&slots[lane].J));
                    }
                    // minimum over the team: by key, or in best-of-K mode by (step, J, k)
                    const uint32_t ka = best_mode ? (kk == kNoKey ? kNoKey : kk >> 10) : kk;
                    uint32_t amin = ka;
    #pragma unroll
                    for (int o = 16; o > 0; o >>= 1) amin = min(amin, __shfl_xor_sync(0xFFFFFFFFu, amin, o));
                    unsigned long long jmin = ka == amin ? jb : ~0ull;
    #pragma unroll
                    for (int o = 16; o > 0; o >>= 1) jmin = min(jmin, __shfl_xor_sync(0xFFFFFFFFu, jmin, o));
                    uint32_t kmin = (ka == amin && jb == jmin) ? kk : kNoKey;
    #pragma unroll
                    for (int o = 16; o > 0; o >>= 1) kmin = min(kmin, __shfl_xor_sync(0xFFFFFFFFu, kmin, o));
                    if (kmin != kNoKey && kk == kmin) {           // keys are unique: exactly one lane
                        const TeamSlot* src = slots + lane;
                        MoveRec& m = sh.rec;
                        m.key = kmin; m.a = __ldcg(&src->a); m.b = __ldcg(&src->b); m.pq = __ldcg(&src->pq);
                        m.J = __ldcg(&src->J);
                        m.d[0] = __ldcg(&src->d[0]); m.d[1] = __ldcg(&src->d[1]); m.d[2] = __ldcg(&src->d[2]);
                    }
                    if (lane == 0) sh.team_key = kmin;
                }
                __syncthreads();
                key_best = sh.team_key;
                ++tw;
            } else if (key_best != kNoKey) {
                const uint32_t owner_lane_mask = __ballot_sync(0xFFFFFFFFu, win_key == key_best);
                if (owner_lane_mask != 0u && lane == __ffs((int)owner_lane_mask) - 1) {
                    MoveRec& m = sh.rec;
                    m.key = key_best; m.a = win_a; m.b = win_b; m.pq = win_pq; m.J = win_J;
                    m.d[0] = win_d0; m.d[1] = win_d1; m.d[2] = win_d2;
                }
                __syncthreads();
            }
            const MoveRec* mv = &sh.rec;

            // ---- commit: null counts of the committed steps, then the move (D9.4)
            steps_done = key_best != kNoKey ? (key_best >> 10) + 1u : Wc;
            {
                const uint32_t lim = steps_done * (uint32_t)K;       // candidates c < lim are committed
                const uint32_t n_comm = gtid < lim ? (lim - 1u - gtid) / GT + 1u : 0u;
#pragma unroll
                for (int wd = 0; wd < kNullWords; ++wd) {
                    const uint32_t lo = 32u * (uint32_t)wd;
                    if (n_comm > lo)
                        my_null += __popc(n_comm >= lo + 32u ? nullw[wd] : (nullw[wd] & ((1u << (n_comm - lo)) - 1u)));
                }
            }
            if (key_best != kNoKey) {
                apply_move(mv, key_best & 1023u, t0 + (key_best >> 10));
                if (hist_valid) { hist_pending = true; hist_a = mv->a; hist_b = mv->b; }
                W = min(steps_done, w_cap);                         // the observed gap (a quarter of the gap between moves
                                                                    // was tried: no gain on c4, 3-6 % slower on the chain sweep)
                depth = 0;
            } else {
                W = min(W * 2u, w_cap);                             // (doubling only once depth >= 4 W, to waste less after a
                                                                    // move, was tried: per-window costs outweigh it, 1-16 chains 10-30 % slower)
                depth += steps_done;
            }
            ++it;
        }
        t0 += steps_done;


        // ---- mode switches (R > 1): every block of the team takes the same decision from the same history
        if (R > 1 && t0 < t_end) {
            if (team) {
                if (key_best != kNoKey && (unsigned long long)steps_done * (unsigned)K < (unsigned long long)AA.team_off) {
                    set_mode(false);                            // followers go and wait at the top of the loop
                    hist_valid = false; hist_pending = false;
                    W = min(W, w_cap);
                }
            } else if ((unsigned long long)W * (unsigned)K >= (unsigned long long)AA.team_on) {
                // leader: windows have grown -> write the state back, call the team
                store_state();
                __syncthreads();
                if (tid == 0) {
                    ctl->W = W; ctl->t0 = t0; ctl->J = sh.J; ctl->depth = depth;
                    __threadfence();
                    st_release_u32(&ctl->phase_seq, phase + 1u);
                }
                ++phase;
                set_mode(true);
            }
        }
    }

    // ---- epilogue: release waiting followers, write back (rank 0 owns the global copy; nulls are summed over blocks)
    if (R > 1 && rank == 0 && !team) {
        __syncthreads();
        if (tid == 0) {
            ctl->W = 1; ctl->t0 = t_end; ctl->J = sh.J; ctl->depth = depth;
            __threadfence();
            st_release_u32(&ctl->phase_seq, phase + 1u);
        }
    }
    if (my_null) atomicAdd(&sh.n_null, my_null);
    __syncthreads();
    if (rank == 0) {
        store_state();
        if (tid == 0) {
            g_stats[0] = sh.n_accept;
            g_stats[2] = sh.hash;
            g_stats[3] = sh.last_accept;
            g_stats[4] = (unsigned long long)__double_as_longlong(sh.J);
            if (AA.depth_all) AA.depth_all[chain_local] = depth;
            if (AA.steps_done_all) AA.steps_done_all[chain_local] = t0 - A.step0;
        }
    }
    if (tid == 0 && sh.n_null) atomicAdd(&g_stats[1], sh.n_null);
}

constexpr int kPartLat = HEA_MC2_PART & 1;
constexpr bool kPartBest = (HEA_MC2_PART >> 1) != 0;

template <int M, int OCC, bool SYM>
cudaError_t launch2_one(const KParams& P, const DevTables& host_tab, const Mc2Args& AA, int64_t C, int threads, size_t smem,
                        cudaStream_t st)
{
    McConst<M> Kc;
    for (int s = 0; s < 3; ++s)
        for (int i = 0; i < M * M; ++i) {
            Kc.g[s * M * M + i] = s < P.S ? host_tab.g[s * M * M + i] : 0.0;
            Kc.t[s * M * M + i] = s < P.S ? host_tab.t[s * M * M + i] : 0.0;
        }
    for (int s = 0; s < 4; ++s) Kc.w[s] = host_tab.w[s];
    auto kern = mc_halo_kernel<M, OCC, SYM, kPartLat, kPartBest>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(C * AA.a.R));
    cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;            // teams spin on each other: all blocks must be co-resident
    attr[0].val.cooperative = AA.a.R > 1 ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, P, Kc, AA);
}

template <int M>
cudaError_t launch2_m(bool sym, int occ_mode, const KParams& P, const DevTables& host_tab, const Mc2Args& AA, int64_t C,
                      int threads, size_t smem, cudaStream_t st)
{
    if (occ_mode == OCC2_NIB) {
        if (M > 4) return cudaErrorInvalidValue;            // a nibble holds a one-hot code of at most 4 species
        constexpr int MN = M > 4 ? 4 : M;
        return sym ? launch2_one<MN, OCC2_NIB, true>(P, host_tab, AA, C, threads, smem, st)
                   : launch2_one<MN, OCC2_NIB, false>(P, host_tab, AA, C, threads, smem, st);
    }
    return sym ? launch2_one<M, OCC2_U8, true>(P, host_tab, AA, C, threads, smem, st)
               : launch2_one<M, OCC2_U8, false>(P, host_tab, AA, C, threads, smem, st);
}

}  // namespace

#define HEA_MC2_CAT2(a, b) a##b
#define HEA_MC2_CAT(a, b) HEA_MC2_CAT2(a, b)
// this part's entry: AA points to an Mc2Args (same layout in every part)
cudaError_t HEA_MC2_CAT(launch_mc2_part, HEA_MC2_PART)(bool sym, int occ_mode, const KParams& P, const DevTables& host_tab,
                                                       const void* AA_, int64_t C, int threads, size_t smem, cudaStream_t st)
{
    const Mc2Args& AA = *reinterpret_cast<const Mc2Args*>(AA_);
    switch (P.M) {
        case 1: return launch2_m<1>(sym, occ_mode, P, host_tab, AA, C, threads, smem, st);
        case 2: return launch2_m<2>(sym, occ_mode, P, host_tab, AA, C, threads, smem, st);
        case 3: return launch2_m<3>(sym, occ_mode, P, host_tab, AA, C, threads, smem, st);
        case 4: return launch2_m<4>(sym, occ_mode, P, host_tab, AA, C, threads, smem, st);
        case 5: return launch2_m<5>(sym, occ_mode, P, host_tab, AA, C, threads, smem, st);
        case 6: return launch2_m<6>(sym, occ_mode, P, host_tab, AA, C, threads, smem, st);
        case 7: return launch2_m<7>(sym, occ_mode, P, host_tab, AA, C, threads, smem, st);
        default: return launch2_m<8>(sym, occ_mode, P, host_tab, AA, C, threads, smem, st);
    }
}

#if HEA_MC2_PART == 0
cudaError_t launch_mc2_part1(bool, int, const KParams&, const DevTables&, const void*, int64_t, int, size_t, cudaStream_t);
cudaError_t launch_mc2_part2(bool, int, const KParams&, const DevTables&, const void*, int64_t, int, size_t, cudaStream_t);
cudaError_t launch_mc2_part3(bool, int, const KParams&, const DevTables&, const void*, int64_t, int, size_t, cudaStream_t);

// Shared-memory bytes of the halo engine (occ_mode 1 = one-hot bytes, 2 = one-hot nibbles).
size_t mc2_shared_bytes(int occ_mode, int lattice, const int* L, int M)
{
    const int A = lattice == 0 ? 4 : 2;
    const size_t NP = (size_t)(L[0] + 2) * (L[1] + 2) * (L[2] + 2) * A;
    size_t s = ((occ_mode == OCC2_NIB ? (NP + 1) / 2 : NP) + 15) & ~(size_t)15;
    s += (sizeof(Sh2) + 15) & ~(size_t)15;
    s += sizeof(int) * (size_t)A * (lattice == 0 ? zpad<0>() : zpad<1>());
    s += (sizeof(float) * (size_t)M * M * filt_row(M) + 15) & ~(size_t)15;       // reject-filter table
    return (s + 15) & ~(size_t)15;
}

size_t mc2_team_bytes(int64_t C) { return sizeof(TeamCtl) * (size_t)C; }

cudaError_t launch_mc2(const KParams& P, const DevTables& host_tab, int lattice, int occ_mode, int threads, int team,
                       void* team_ctl, int team_on, int team_off, int accept_engine, size_t smem_budget, int w_max, uint8_t* occ, int32_t* counts, int64_t C, uint64_t n_steps, int K, uint64_t seed, uint64_t chain0,
                       uint64_t step0, void* stats, void* log, int64_t log_cap, int select_best, uint64_t depth_limit,
                       uint64_t* depth, uint64_t* steps_done, uint32_t* hist, cudaStream_t st, int64_t* n_launches)
{
    Mc2Args AA;
    McArgs& A = AA.a;
    A.occ_all = occ; A.counts_all = counts;
    A.n_steps = n_steps; A.seed = seed; A.chain0 = chain0; A.step0 = step0;
    A.stats_all = reinterpret_cast<unsigned long long*>(stats);
    A.log_all = reinterpret_cast<unsigned long long*>(log);
    A.log_cap = log_cap; A.K = K; A.R = team; A.w_max = w_max; A.fast_nbr = 0;
    AA.team = reinterpret_cast<TeamCtl*>(team_ctl);
    AA.team_on = team_on > 0 ? team_on : 4 * threads;
    AA.team_off = team_off > 0 ? team_off : threads;
    AA.accept_engine = accept_engine;
    AA.hist = hist;
    AA.select_best = select_best ? 1 : 0;
    AA.depth_limit = depth_limit;
    AA.depth_all = reinterpret_cast<unsigned long long*>(depth);
    AA.steps_done_all = reinterpret_cast<unsigned long long*>(steps_done);
    if (team > 1) {
        if (team > kMaxTeam || !team_ctl) return cudaErrorInvalidValue;
        cudaError_t em = cudaMemsetAsync(team_ctl, 0, mc2_team_bytes(C), st);
        if (em != cudaSuccess) return em;
    }
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
    Geo& G = AA.G;
    for (int d = 0; d < 3; ++d) G.L[d] = P.L[d];
    auto magic = [](int d) { return d == 1 ? 0xFFFFFFFFu : (uint32_t)((1ull << 32) / (uint64_t)d); };
    // exact division of n < 2^31 by d >= 2: with l = ceil(log2 d), s = l - 1 and m = ceil(2^(32+s) / d) < 2^32 the error
    // e = m d - 2^(32+s) is < d <= 2^l, so n e < 2^(32+s) and floor(n m / 2^(32+s)) = floor(n / d)
    auto div_magic = [](uint64_t d, uint32_t& m, uint32_t& sft) {
        int l = 0;
        while ((1ull << l) < d) ++l;
        sft = (uint32_t)(l - 1);
        m = (uint32_t)(((1ull << (32 + sft)) + d - 1) / d);
    };
    {
        // the floor keeps the rounding of the D6 evaluation (absolute error ~ 2^-53 A per cell, A = |x| + |1-x| + |d|
        // <= 2 / c_min + 2 + |t|) below 0.05 % of a first-shell term that reaches the threshold
        double inv_c_max = 1.0, t_max = 0.0;
        for (int i = 0; i < P.M; ++i) {
            inv_c_max = std::max(inv_c_max, std::sqrt((double)P.N * (double)P.z[0] * host_tab.g[i * P.M + i]));
            for (int j = 0; j < P.M; ++j) t_max = std::max(t_max, std::fabs(host_tab.t[i * P.M + j]));
        }
        const double Amax = 2.0 * inv_c_max + 2.0 + t_max;
        AA.filt_floor = 1.0e-18 * host_tab.w[0] * std::max(1.0, (Amax / 100.0) * (Amax / 100.0));
    }
    AA.k_mq = 0u; AA.k_sq = 0u;
    if (K >= 2) div_magic((uint64_t)K, AA.k_mq, AA.k_sq);
    div_magic((uint64_t)P.A * (uint64_t)P.L[2], G.mq, G.sq);
    div_magic((uint64_t)P.A * (uint64_t)P.L[1] * (uint64_t)P.L[2], G.mx, G.sx);
    G.PLy = P.L[1] + 2; G.PLz = P.L[2] + 2;
    G.cx = (uint32_t)(2 * P.A * G.PLz);
    G.cc = (uint32_t)(P.A * (G.PLy * G.PLz + G.PLz + 1));
    G.pmagy = magic(G.PLy); G.pmagz = magic(G.PLz);
    G.NP = (P.L[0] + 2) * G.PLy * G.PLz * P.A;
    {
        // first-shell decomposition (see Mc2Args): groups = vectors with the same neighbour basis seen from basis 0
        const int A = P.A, Z = P.Z, z0 = P.z[0];
        auto off = [&](int b, int k) {
            const int8_t* stn = host_tab.stencil + (b * Z + k) * 4;
            return (((int)stn[1] * G.PLy + (int)stn[2]) * G.PLz + (int)stn[3]) * A + ((int)stn[0] - b);
        };
        int order[24], n_ord = 0;
        for (int nb = 0; nb < A; ++nb)
            for (int k = 0; k < z0; ++k)
                if (host_tab.stencil[(0 * Z + k) * 4] == nb) order[n_ord++] = k;
        if (n_ord != z0 || z0 > 12 || (z0 & 3)) return cudaErrorInvalidValue;
        for (int i = 0; i < 12; ++i) AA.fs_c[i] = 0;
        for (int b = 0; b < 4; ++b) for (int g = 0; g < 4; ++g) AA.fs_rd[b][g] = 0;
        for (int i = 0; i < z0; ++i) {
            const int k = order[i], nb0 = host_tab.stencil[(0 * Z + k) * 4];
            const int c = off(0, k) - nb0;                   // A * (cell part): even
            if (c & 1) return cudaErrorInvalidValue;
            AA.fs_c[i] = occ_mode == OCC2_NIB ? c / 2 : c;
            for (int b = 0; b < A; ++b) {
                const int rd = off(b, k) - c;
                if ((i & 3) == 0) AA.fs_rd[b][i >> 2] = rd;
                else if (AA.fs_rd[b][i >> 2] != rd) return cudaErrorInvalidValue;      // not of the assumed form
            }
        }
    }
    for (int r = 0; r < 10; ++r) {
        AA.rk[2 * r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u;
        AA.rk[2 * r + 1] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
    }
    if (lattice == 0) { G.basis = (1u << 4) | (1u << 5) | (1u << 6) | (1u << 8) | (1u << 9) | (1u << 10); G.d2[0] = 2; G.d2[1] = 4; G.d2[2] = 6; }
    else { G.basis = (1u << 3) | (1u << 4) | (1u << 5); G.d2[0] = 3; G.d2[1] = 4; G.d2[2] = 8; }
    G.distinct = P.L[0] >= 3 && P.L[1] >= 3 && P.L[2] >= 3;
    size_t smem = mc2_shared_bytes(occ_mode, lattice, P.L, P.M);
    // the pipelined accept engine needs its record, bitmap and offset buffers on top; without room it is simply off
    auto pae_bytes_of = [&](int ds) {
        const size_t dwords = ((((size_t)P.N + ((size_t)1 << ds) - 1) >> ds) + 31) >> 5;
        return sizeof(PRec) * (size_t)kPaeRecs + 4u * dwords + 4u * (size_t)P.A * (size_t)P.Z + 16u +
               8u * 2u * (size_t)kPaeK * (size_t)P.S * (size_t)P.M + 8u + sizeof(uint2) * (size_t)kPaeRecs;
    };
    // The site-histogram filter is bound by the random L2 loads an SM can keep in flight, and those need L1 lines: with the
    // 228 KB shared-memory carve-out (28 KB of L1) an SM sustains ~0.5 random sectors per clock, with 196 KB ~0.9.  When the
    // table is in use, the touched-site bitmap of the accept engine is made coarser (conservative) if that brings the block
    // under the 196 KB carve-out (1 KB of it is reserved by the system).
    AA.dshift = 0;
    if (hist != nullptr && accept_engine == 2 && threads >= 512) {
        const size_t target = 196u * 1024u - 1024u;
        for (int ds = 0; ds <= 4; ++ds)
            if (smem + pae_bytes_of(ds) <= target) { AA.dshift = ds; break; }
    }
    const size_t pae_bytes = pae_bytes_of(AA.dshift);
    AA.pae = (accept_engine == 2 && threads >= 512 && smem + pae_bytes <= smem_budget) ? 1 : 0;
    if (AA.pae) smem += pae_bytes;
    const int part = (lattice != 0 ? 1 : 0) + (select_best ? 2 : 0);
    cudaError_t e = part == 0 ? launch_mc2_part0(sym, occ_mode, P, host_tab, &AA, C, threads, smem, st)
                  : part == 1 ? launch_mc2_part1(sym, occ_mode, P, host_tab, &AA, C, threads, smem, st)
                  : part == 2 ? launch_mc2_part2(sym, occ_mode, P, host_tab, &AA, C, threads, smem, st)
                              : launch_mc2_part3(sym, occ_mode, P, host_tab, &AA, C, threads, smem, st);
    if (e == cudaSuccess) ++*n_launches;
    return e;
}

#endif  // HEA_MC2_PART == 0

}  // namespace hea
