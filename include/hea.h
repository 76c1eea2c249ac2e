/*
 * hea.h -- C ABI of libhea_b200: the data-parallel hot path of PyHEA (arxiv 2411.18906) on NVIDIA B200 (sm_100a).
 *
 * The path (citations "P:<n>" = PAPER.md line; "D<n>/A<n>" = DESIGN.md section 3):
 *   hea_create        lattice supercell S = A*L^3, species concentrations, coordination shells,
 *                     shell weights w_k and target alpha; builds the shell neighbour tables on the host (D1-D3)
 *   hea_init_random   seeded exact-composition random start (D8)
 *   hea_sro_full      full Warren-Cowley recount: ordered pair counts N_ij^(k), alpha_ij^(k) = 1 - P_ij^(k)/c_j (Eq. 2,
 *                     P:256-262) and J = F^2 = sum_k w_k sum_ij (alpha - alpha_target)^2 (Eq. 3)  (D4-D6)
 *   hea_mc_run        chain-parallel Monte Carlo local search (Alg. 3): per step K candidate swaps, each
 *                     evaluated by the incremental pair-count update (Eq. 4; Eq. 5), the
 *                     lowest-index improving candidate applied (D9)
 *   hea_mc_run_ex     the same with the paper's own selection and termination: best-of-K (Eq. 6) and the
 *                     search-depth counter (Alg. 3)  (A23)
 *   hea_pool_select   selection step of the global search (Alg. 1)  (A24)
 *   hea_pool_rank_static  its ranking step with no device allocation (static scratch of a fixed size)
 *
 * Conventions for every call
 *   - All functions return HEA_OK (0) or an error code; hea_last_error() gives a thread-local message.
 *   - Pointers named *_dev are DEVICE pointers on the context's device, owned by the caller (e.g. torch tensors);
 *     pointers named *_host are HOST pointers owned by the caller.  The library owns only hea_ctx and its tables.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device entry points are
 *     asynchronous on that stream: argument errors are reported synchronously before any launch; device faults
 *     surface at the caller's next synchronisation.  *_host entry points are synchronous.
 *   - Layouts are dense, row-major, little-endian: occ [C][N] uint8 (species id < n_species; larger values are
 *     undefined behaviour, not validated on the hot path), counts [C][S][M][M] int32, alpha [C][S][M][M] double.
 *   - Site order (D1): site = ((x*Ly + y)*Lz + z)*A + b with basis fcc A=4 (0,0,0),(0,1,1),(1,0,1),(1,1,0),
 *     bcc A=2 (0,0,0),(1,1,1) in units of a/2.  Shells (D2): fcc |o|^2 = 2,4,6 (z = 12,6,24), bcc 3,4,8 (z = 8,6,12),
 *     offsets in lexicographic order, periodic; tiny cells keep exactly z_s table entries (multi-edge semantics).
 *   - Empty batches (B == 0 / C == 0) return HEA_OK without touching the buffers (their pointers may be NULL).
 *   - There is no CPU fallback: without a CUDA device every compute call returns HEA_ECUDA.
 *   - One context serves ONE stream and ONE host thread at a time: the context owns scratch buffers (team control
 *     blocks of hea_mc_run, the pool buffers of hea_pool_select, the staging buffers of the *_host calls) that are
 *     reused by every call.  Calls on the same stream are ordered and safe; before using a context from another stream
 *     or thread, or before a *_host call that follows asynchronous calls, synchronise the previous stream.  Use one
 *     context per stream for concurrent work (contexts share nothing).
 *   - Limits checked by hea_create: n_species in [1, 8], n_shells in [1, 3], every L >= 1, N < 2^31 and
 *     max_s(z_s) * N < 2^31 (the ordered pair counts are int32), finite shell weights and targets.  Negative shell
 *     weights are accepted (J may then be negative; lower-bound pruning and the reduced-precision filter switch off).
 */
#ifndef HEA_H
#define HEA_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hea_ctx hea_ctx;                 /* opaque; created by hea_create, freed by hea_destroy */

enum { HEA_FCC = 0, HEA_BCC = 1 };
enum { HEA_OK = 0, HEA_EINVAL = 1, HEA_EUNSUPPORTED = 2, HEA_ENOMEM = 3, HEA_ECUDA = 4 };

#define HEA_MAX_SPECIES 8
#define HEA_MAX_SHELLS  3
#define HEA_MAX_K       1024
#define HEA_HASH_INIT   0xcbf29ce484222325ULL   /* initial value of hea_mc_stats.hash (D9.4) */
#define HEA_NO_STEP     0xffffffffffffffffULL   /* initial value of hea_mc_stats.last_accept_step */

/* Per-chain running statistics of hea_mc_run (in/out: counters and hash continue across calls; J is output). */
typedef struct {
    uint64_t n_accept;           /* accepted moves */
    uint64_t n_null;             /* candidate slots that stayed like-species after the one redraw (D9.1) */
    uint64_t hash;               /* FNV-1a style hash over (step lo, step hi, k, a, b) of every accepted move */
    uint64_t last_accept_step;   /* absolute step of the last accepted move, HEA_NO_STEP if none */
    double   J;                  /* objective J = F^2 of the current configuration (D6) */
} hea_mc_stats;

/* One accepted move. */
typedef struct { uint64_t step; uint32_t k, a, b; } hea_move;

/* Library version string (static storage). */
const char* hea_version(void);

/* Thread-local message of the last error returned on this thread (static storage, never NULL). */
const char* hea_last_error(void);

/*
 * hea_create -- problem statement of the paper: P:105 (lattice, supercell), P:35/P:142 (species, concentrations),
 * P:271 (shells, weights w_k, target alpha).
 *   lattice          HEA_FCC | HEA_BCC;  Lx,Ly,Lz >= 1 conventional cells;  N = A*Lx*Ly*Lz < 2^31
 *   conc             [n_species] host, > 0, sums to 1 within 1e-9; species counts N_i by D3 (round if integral,
 *                    else floor + largest remainder, ties to the lower index); any N_i == 0 -> HEA_EINVAL
 *   shell_w          [n_shells] host;  alpha_target [n_shells][n_species][n_species] host, row-major
 *   n_species in [1, 8], n_shells in [1, 3] (else HEA_EUNSUPPORTED)
 *   device           CUDA device ordinal.  Builds the device neighbour table (site-major [N][Z], rows padded to
 *                    whole 32-site tiles; shared by the recount and the MC kernel).
 * All host arrays are copied.  Errors: HEA_EINVAL, HEA_EUNSUPPORTED, HEA_ENOMEM, HEA_ECUDA (no device / alloc failed).
 */
int hea_create(hea_ctx** out, int lattice, int Lx, int Ly, int Lz,
               int n_species, const double* conc,
               int n_shells, const double* shell_w, const double* alpha_target,
               int device);

/* Frees the context and its device tables.  NULL is allowed. */
int hea_destroy(hea_ctx* ctx);

/* n_sites, z[n_shells], n_per_species[n_species] (any output pointer may be NULL). */
int hea_info(const hea_ctx* ctx, int64_t* n_sites, int* z, int64_t* n_per_species);

/* Host copy of the shell's neighbour table, [N][z_shell] int32, entry k = site at offset o_k (D2).  For tests. */
int hea_neighbor_table(const hea_ctx* ctx, int shell, int32_t* out_host);

/*
 * Tuning knobs (never change results).  name:
 *   "mc_occ_mode"     0 = auto, 1 = shared uint8, 2 = shared 4-bit packed, 3 = global memory (through L2)
 *   "mc_threads"      threads per block: 0 = auto, else a multiple of 32 in [32, 1024]
 *   "mc_cluster"      blocks per chain (thread-block cluster, replicated chain state): 0 = auto, 1..8
 *   "mc_window"       cap on the speculative step window (steps evaluated against one configuration before the
 *                     lowest improving (step, k) is applied): 0 = auto, 1 = strictly step by step, up to 2^20
 *   "mc_neighbors"    0 = auto, 1 = always the neighbour table, 2 = interior sites use site + offset (no table load)
 *   "mc_engine"       0 = auto (2 when the padded one-hot configuration fits in shared memory), 1 = table-driven
 *                     window engine (hea_mc.cu), 2 = shared-memory "halo" engine (hea_mc2.cu; HEA_EINVAL if it does not fit)
 *   "mc_team"         halo engine: blocks per chain (replicas synchronised through global memory, cooperative launch),
 *                     0 = auto (min(32, SMs / C)), 1..32;  "mc_team_on" / "mc_team_off": window sizes (candidates) at which
 *                     a team starts / stops sharing a window, 0 = auto
 *   "mc_accept"       halo engine, single-step windows: 0 = auto (3), 1 = thread per candidate, 2 = eight lanes per
 *                     candidate, 3 = the warp-specialised serial engine over epochs of records computed ahead
 *   "mc_hist"         halo engine, long windows: the reject filter reads a per-site table (species and first-shell
 *                     neighbour counts, 4 bytes per site and chain, library-owned, kept in L2) instead of gathering the
 *                     neighbours; 0 = auto (on for 2..5 species on cells of at least 3 cells per side while the tables of
 *                     all chains take at most 64 MB), 1 = off, 2 = on whatever the size
 *   "sro_engine"      recount: 0 = auto (the table-free stencil kernel when occ_dev is aligned to the basis size,
 *                     else the table-driven kernel), 1 = table-driven (HBM-bound, 4 Z + 1 bytes per atom),
 *                     2 = stencil (1 byte per atom; HEA_EINVAL when occ_dev is not aligned)
 *   "sro_tile_xy"     stencil recount: cap on the tile extent along x and y in cells, 0 = auto (8), 1..8
 *   "sro_tile_z"      stencil recount: row pitch of the staged tile, 0 = auto, else 12, 22 or 34 (tiles of up to
 *                     10, 20, 32 cells along z)
 *   "sro_flush_tiles" stencil recount: cap on the tiles a thread accumulates before its packed rows are unpacked,
 *                     0 = auto (what the packed fields hold), 1..2^20
 *   "sro_lanes"       stencil recount: lane mapping, 0 = auto (2), 1 = over the row words incl. the halo (conflict-free
 *                     shared-memory loads, some lanes idle), 2 = over the interior cells only
 *   "sro_threads"     stencil recount: threads per block, 0 = auto, else a multiple of 32 in [128, 384]
 *   "sro_warps"       table recount: warps per block, 0 = auto (16), 1..16
 *   "sro_stages"      table recount: cap on the per-warp ring of 32-site table tiles in shared memory, 0 = auto, 1..8
 *   "sro_blocks_per_sm"  recount (both engines): resident blocks per SM the grid and the shared-memory split are sized for, 0 = auto, 1..4
 * Unknown name or value -> HEA_EINVAL.
 */
int hea_set_option(hea_ctx* ctx, const char* name, int64_t value);
int hea_get_option(const hea_ctx* ctx, const char* name, int64_t* value);

/*
 * hea_init_random -- D8 ("generated entirely randomly"): occ[c] = species blocks in ascending order, then
 * Fisher-Yates for n = N-1..1 with j = (Philox4x32-10(ctr=(n,0,0xFFFFFFFF,chain0+c), key=seed)[0] * (n+1)) >> 32.
 *   occ_dev [C][N] uint8 out;  chain0 + C <= 2^32.
 */
int hea_init_random(hea_ctx* ctx, uint8_t* occ_dev, int64_t C, uint64_t seed, uint64_t chain0, void* cuda_stream);

/*
 * hea_sro_full -- D4-D6 (Eq. 2, Eq. 3): for each of B configurations
 *   counts[s][i][j] = #{(a, k < z_s) : occ[a] = i and occ[nbr_s[a][k]] = j}      (ordered pairs, int32)
 *   alpha[s][i][j]  = 1 - counts * g,  g = N / (z_s N_i N_j)                       (optional, may be NULL)
 *   obj[b]          = J = sum_s w_s sum_i sum_j (alpha - alpha_target)^2           (optional, may be NULL)
 * evaluated in fp64 in the fixed order of D6 (no FMA contraction).  counts_dev is overwritten.
 * Two device engines give the same integers ("sro_engine"): the table-free stencil kernel (default; 1 byte of HBM traffic
 * per atom; needs occ_dev aligned to the basis size, 4 for fcc, 2 for bcc) and the table-driven kernel (4 Z + 1 bytes per
 * atom, HBM-bound; taken automatically for unaligned occ_dev).  Asynchronous on cuda_stream.
 */
int hea_sro_full(hea_ctx* ctx, const uint8_t* occ_dev, int64_t B,
                 int32_t* counts_dev, double* alpha_dev, double* obj_dev, void* cuda_stream);

/* Sets stats_dev[0..C) to {0, 0, HEA_HASH_INIT, HEA_NO_STEP, 0.0}. */
int hea_mc_stats_reset(hea_ctx* ctx, hea_mc_stats* stats_dev, int64_t C, void* cuda_stream);

/*
 * hea_mc_run -- D9 (Alg. 3 P:242-250 with Eq. 4-5): advances C independent chains by n_steps steps.
 * Per chain c (global id chain0 + c < 2^32) and absolute step t = step0 + 0..n_steps-1:
 *   for k = 0..K-1: (r0..r3) = Philox4x32-10(ctr=(t lo, t hi, k, chain), key=seed); a = (r0*N)>>32,
 *   b = (r1*(N-1))>>32, b += (b >= a); if occ[a] == occ[b] redraw once from (r2, r3); still alike -> null candidate.
 *   Every non-null candidate's J_k is computed from counts + delta (neighbours of a and b except a, b themselves)
 *   in the D6 order; the lowest k with J_k < J_cur (strict) is applied: occ swapped, counts updated, stats updated.
 *   occ_dev    [C][N] in/out
 *   counts_dev [C][S][M][M] in/out; MUST equal the recount of occ_dev on entry (get it from hea_sro_full)
 *   stats_dev  [C] in/out (see hea_mc_stats; initialise with hea_mc_stats_reset for a fresh chain)
 *   log_dev    [C][log_cap] accepted moves of THIS call in order (first log_cap of them), or NULL with log_cap 0
 *   K in [1, HEA_MAX_K].  Results depend only on (seed, chain id, step), never on C, batching or tuning options:
 *   run(S1) followed by run(S2, step0 = S1) equals run(S1 + S2).
 *   Arithmetic: int32 counts, fp64 objective in the D6 order.  With a bit-symmetric target and weights >= 0, long windows
 *   first pass a conservative fp32 reject filter on the first shell (the paper's own reduced precision: P:297); its
 *   threshold carries a proven error bound and every survivor is evaluated in fp64, so the accept decisions are exactly
 *   those of the fp64 rule.
 */
int hea_mc_run(hea_ctx* ctx, uint8_t* occ_dev, int32_t* counts_dev, int64_t C, uint64_t n_steps, int K,
               uint64_t seed, uint64_t chain0, uint64_t step0,
               hea_mc_stats* stats_dev, hea_move* log_dev, int64_t log_cap, void* cuda_stream);

/*
 * hea_mc_run_ex -- hea_mc_run with the paper's own selection and termination as options.
 *   select_best != 0: per step the candidate with the smallest J_k is taken (Eq. 6: F_best = min over the
 *                     updates; ties -> lowest k) and applied iff J_k < J_cur; 0: lowest improving k (hea_mc_run).
 *   depth_limit > 0:  search-depth termination (Alg. 3, section 4.6.4): depth = consecutive steps
 *                     without an applied move, reset by every applied move; a chain stops as soon as
 *                     depth == depth_limit (a chain entering with depth >= depth_limit does nothing), else after
 *                     n_steps steps.  0: no depth termination.
 *   depth_dev      [C] uint64 in/out: the depth counters (carry them over for split runs); may be NULL when
 *                  depth_limit == 0
 *   steps_done_dev [C] uint64 out: steps executed by this call (n_steps unless the depth limit stopped the chain);
 *                  may be NULL
 * Everything else as hea_mc_run; hea_mc_run == hea_mc_run_ex(select_best 0, depth_limit 0, NULL, NULL).
 * Returns HEA_EUNSUPPORTED for a non-default option when the configuration does not fit the shared-memory engine.
 */
int hea_mc_run_ex(hea_ctx* ctx, uint8_t* occ_dev, int32_t* counts_dev, int64_t C, uint64_t n_steps, int K,
                  uint64_t seed, uint64_t chain0, uint64_t step0,
                  hea_mc_stats* stats_dev, hea_move* log_dev, int64_t log_cap,
                  int select_best, uint64_t depth_limit, uint64_t* depth_dev, uint64_t* steps_done_dev,
                  void* cuda_stream);

/*
 * hea_pool_select -- the selection step of the global search (Alg. 1; retained top solutions seed the
 * next iteration, the others are generated entirely randomly) over a pool of C chains.
 * The chains are ranked by J of counts_dev (D6), ascending, ties -> lower index.  The n_keep best move to positions
 * 0..n_keep-1 in rank order with their counts and stats; every position r >= n_keep receives a fresh seeded random
 * configuration (hea_init_random, chain id new_chain0 + r - n_keep), its recount, and reset stats.  The paper gives no
 * value for the retained fraction ("at most half") or the discarded fraction p_a: n_keep is the caller's.
 *   occ_dev [C][N], counts_dev [C][S][M][M], stats_dev [C]: in/out; counts_dev must be the recount of occ_dev
 *   order_dev [n_keep] int32 out (optional, may be NULL): previous index of the chain now at each kept position
 * A chain at position r continues with RNG chain id chain0 + r of the next hea_mc_run.  C <= 65,536.
 */
int hea_pool_select(hea_ctx* ctx, uint8_t* occ_dev, int32_t* counts_dev, hea_mc_stats* stats_dev, int64_t C,
                    int64_t n_keep, uint64_t seed, uint64_t new_chain0, int32_t* order_dev, void* cuda_stream);

/*
 * hea_pool_rank_static -- the ranking step of hea_pool_select (Alg. 1; A24) for callers that cannot allocate
 * device memory (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): this call allocates
 * nothing, on the host side of the device or on the device -- no cudaMalloc, cudaFree or allocating library routine.
 *   counts_dev [C][S][M][M] in: the recount of each chain;  order_dev [n_keep] int32 out: order_dev[r] = index of the chain
 *   of rank r by J (D6) ascending, ties -> lower index -- what hea_pool_select(n_keep) reports in its order_dev.
 * Its scratch (J of every chain) is a static device array inside the library of HEA_POOL_RANK_STATIC_MAX doubles
 * (512 KB) that every GPU loading the library holds until the process exits.  C > HEA_POOL_RANK_STATIC_MAX -> HEA_EINVAL
 * with a message naming the limit (hea_pool_select has no such limit below 65,536 but allocates).
 * The array is shared by EVERY call in the process, whatever the context, and keeps the last call's contents; this
 * call overwrites the entries it reads, so nothing needs clearing.  Calls that overlap on one GPU (different streams,
 * contexts or threads) race on it: order them on one stream or synchronise between them.  The first call on a device
 * resolves the array's device address (cudaGetSymbolAddress; not an allocation).  Asynchronous on cuda_stream.
 */
#define HEA_POOL_RANK_STATIC_MAX 65536
int hea_pool_rank_static(hea_ctx* ctx, const int32_t* counts_dev, int64_t C, int64_t n_keep, int32_t* order_dev,
                         void* cuda_stream);

/*
 * Host-buffer (end-to-end) forms: the same kernels, with host<->device copies done by the library on an internal
 * stream, synchronous.  Host buffers may be pageable or pinned.
 *   hea_sro_full_host: occ_host [B][N] -> counts_host (required), alpha_host / obj_host (optional).
 *   hea_mc_run_host:   occ_host [C][N] in/out; the library recounts occ on the device first (so no counts input),
 *                      runs hea_mc_run, and returns occ, counts_host [C][S][M][M] (optional) and stats_host [C]
 *                      (in/out, required).
 */
int hea_sro_full_host(hea_ctx* ctx, const uint8_t* occ_host, int64_t B,
                      int32_t* counts_host, double* alpha_host, double* obj_host);
int hea_mc_run_host(hea_ctx* ctx, uint8_t* occ_host, int32_t* counts_host, int64_t C, uint64_t n_steps, int K,
                    uint64_t seed, uint64_t chain0, uint64_t step0, hea_mc_stats* stats_host);

/* Number of kernel launches issued by this context since creation (for bench.py's gpu_launches). */
int hea_launch_count(const hea_ctx* ctx, int64_t* n);

/*
 * hea_measure_peaks -- micro-benchmarks of the resources the kernels of this library are bound by, for the roofline
 * denominators that a copy / GEMM benchmark does not give.  Not part of the method: measurement support
 * for bench.py.  Runs on `cuda_stream` of the context's device and synchronises on it (about 0.3 s).
 * out_host [HEA_N_PEAKS] (HOST, doubles), whole-chip rates:
 *   [0] random shared-memory byte gathers per second (LDS.U8, 32 lanes at random banks of a 128 KB array)
 *   [1] conflict-free shared-memory wavefronts per second (LDS.32, lane l -> bank l)
 *   [2] INT32 ALU-pipe thread-instructions per second (independent LOP3 chains)
 *   [3] FMA-pipe integer thread-instructions per second (independent IMAD chains)
 *   [4] thread-instructions per second with both pipes busy (LOP3 and IMAD interleaved): the issue ceiling
 *   [5] fp64 thread-instructions per second (independent DMUL + DADD chains, no FMA, as in D6)
 *   [6] GB/s of random 32-byte sectors read through L2 (64 MB array)
 *   [7] SM clock in MHz reported by the device attribute
 * Errors: HEA_EINVAL (NULL, n_out < HEA_N_PEAKS), HEA_ENOMEM / HEA_ECUDA.
 */
#define HEA_N_PEAKS 8
int hea_measure_peaks(hea_ctx* ctx, double* out_host, int n_out, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* HEA_H */
