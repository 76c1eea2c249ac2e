/*
 * hea_oracle.c -- plain, slow, obviously-correct CPU ORACLE for the PyHEA hot path
 * (arxiv 2411.18906; citations "P:<n>" are /root/reference/PAPER.md line numbers,
 * "D<n>"/"A<n>" are the definitions / readings listed in DESIGN.md section 3).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or constant with the CUDA library under paper_2411_18906_b200/csrc/.
 *
 * What it computes, in the paper's order:
 *   - the bcc/fcc supercell and its coordination-shell neighbour table     (D1-D2)
 *   - Warren-Cowley alpha_ij^(k) = 1 - P_ij^(k)/c_j from ordered pair counts (Eq. 2; D4-D5)
 *   - the fitness F = sqrt(J), J = sum_k w_k sum_ij (alpha - alpha_target)^2  (Eq. 3; D5-D6)
 *   - the parallel Monte Carlo local search of Alg. 3 in the variant
 *     BASELINE.json:north_star fixes: K candidate swaps per step, all evaluated against
 *     the same x_curr, incremental pair-count deltas (Eq. 4), objective
 *     recomputed from the integer counts (Eq. 5, P:300-307 read as D6/A15), the
 *     lowest-index improving candidate applied                               (D9)
 *   - Philox4x32-10 (Salmon et al., SC'11) keyed by (seed; step, k, chain)  (D7)
 *   - seeded Fisher-Yates initial placement ("generated entirely randomly"; D8)
 *
 * Everything is a direct loop over the definition: no blocking, fusion, packing or
 * reordering.  Floating point is fp64, one rounding per operation (build with
 * -ffp-contract=off, never -ffast-math).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Random123 known-answer vectors for
 * Philox; O(N^2) minimum-image distance search for the table; B2 / L1_2 / L1_0 closed
 * forms for alpha; sum rules; exact-composition shuffle expectation E[alpha]; delta ==
 * recount difference for all unlike pairs on tiny cells; brute-force enumeration of all
 * C(16,8) configurations of a 16-site bcc cell; exhaustive re-evaluation of the
 * lowest-index-improving rule with full recounts.  No function here is "parity unpinned".
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#include <pthread.h>

#define ORA_MAX_SHELLS 3
#define ORA_MAX_SPECIES 8
#define ORA_MAX_Z 24

typedef struct {
    int lattice;               /* 0 = fcc, 1 = bcc */
    int L[3];                  /* conventional cells along x, y, z */
    int A;                     /* basis atoms per conventional cell: 4 fcc, 2 bcc */
    int64_t N;                 /* number of sites = A*Lx*Ly*Lz */
    int M;                     /* species */
    int S;                     /* shells */
    int z[ORA_MAX_SHELLS];     /* neighbours per shell */
    int64_t n_per_species[ORA_MAX_SPECIES];
    double w[ORA_MAX_SHELLS];
    double t[ORA_MAX_SHELLS][ORA_MAX_SPECIES][ORA_MAX_SPECIES];   /* alpha target */
    double g[ORA_MAX_SHELLS][ORA_MAX_SPECIES][ORA_MAX_SPECIES];   /* N/(z_s N_i N_j), D5-D6 */
    int32_t *nbr[ORA_MAX_SHELLS];                                 /* [N][z_s] */
} ora_sys;

typedef struct { uint64_t n_accept, n_null, hash, last_accept_step; double J; } ora_stats;
typedef struct { uint64_t step; uint32_t k, a, b; } ora_move;

/* ---------------------------------------------------------------- D1: lattice */
static const int FCC_BASIS[4][3] = {{0,0,0},{0,1,1},{1,0,1},{1,1,0}};
static const int BCC_BASIS[2][3] = {{0,0,0},{1,1,1}};

static const int (*basis_of(int lattice))[3] { return lattice == 0 ? FCC_BASIS : BCC_BASIS; }

/* position of a site in doubled integer coordinates (unit a/2) */
static void site_position(const ora_sys *sy, int64_t site, int p[3])
{
    int b = (int)(site % sy->A);
    int64_t cell = site / sy->A;
    int zc = (int)(cell % sy->L[2]); cell /= sy->L[2];
    int yc = (int)(cell % sy->L[1]); cell /= sy->L[1];
    int xc = (int)cell;
    const int (*bs)[3] = basis_of(sy->lattice);
    p[0] = 2*xc + bs[b][0]; p[1] = 2*yc + bs[b][1]; p[2] = 2*zc + bs[b][2];
}

/* inverse of site_position for a position already reduced into the box; -1 if not a lattice point */
static int64_t site_of_position(const ora_sys *sy, const int p[3])
{
    const int (*bs)[3] = basis_of(sy->lattice);
    for (int b = 0; b < sy->A; b++) {
        int d0 = p[0]-bs[b][0], d1 = p[1]-bs[b][1], d2 = p[2]-bs[b][2];
        if (d0 < 0 || d1 < 0 || d2 < 0) continue;
        if ((d0 & 1) || (d1 & 1) || (d2 & 1)) continue;
        int xc = d0/2, yc = d1/2, zc = d2/2;
        if (xc >= sy->L[0] || yc >= sy->L[1] || zc >= sy->L[2]) continue;
        return (((int64_t)xc*sy->L[1] + yc)*sy->L[2] + zc)*sy->A + b;
    }
    return -1;
}

/* is the displacement o (doubled coordinates) a lattice vector of the Bravais lattice? */
static int is_lattice_vector(int lattice, int ox, int oy, int oz)
{
    if (lattice == 0)          /* fcc: all integers with even sum */
        return ((ox + oy + oz) & 1) == 0;
    /* bcc: all even or all odd */
    return ((ox & 1) == (oy & 1)) && ((oy & 1) == (oz & 1));
}

/* ---------------------------------------------------------------- D2: shells + table */
/* Fills offs[s][k][3] for the S smallest non-zero squared lengths, offsets lexicographically ascending. */
static void shell_offsets(int lattice, int S, int z[ORA_MAX_SHELLS], int offs[ORA_MAX_SHELLS][ORA_MAX_Z][3])
{
    const int R = 4;           /* |o|^2 <= 8 for the three shells of both lattices; searched, not assumed */
    int d2s[ORA_MAX_SHELLS]; int found = 0; int last = 0;
    while (found < S) {        /* s-th smallest non-zero squared distance */
        int best = 1 << 30;
        for (int ox = -R; ox <= R; ox++) for (int oy = -R; oy <= R; oy++) for (int oz = -R; oz <= R; oz++) {
            if (!is_lattice_vector(lattice, ox, oy, oz)) continue;
            int d2 = ox*ox + oy*oy + oz*oz;
            if (d2 > last && d2 < best) best = d2;
        }
        d2s[found++] = best; last = best;
    }
    for (int s = 0; s < S; s++) {
        int k = 0;
        for (int ox = -R; ox <= R; ox++) for (int oy = -R; oy <= R; oy++) for (int oz = -R; oz <= R; oz++) {
            if (!is_lattice_vector(lattice, ox, oy, oz)) continue;
            if (ox*ox + oy*oy + oz*oz != d2s[s]) continue;
            offs[s][k][0] = ox; offs[s][k][1] = oy; offs[s][k][2] = oz; k++;   /* loop order == lexicographic */
        }
        z[s] = k;
    }
}

static int posmod(int a, int m) { int r = a % m; return r < 0 ? r + m : r; }

static int build_tables(ora_sys *sy)
{
    int offs[ORA_MAX_SHELLS][ORA_MAX_Z][3];
    shell_offsets(sy->lattice, sy->S, sy->z, offs);
    for (int s = 0; s < sy->S; s++) {
        sy->nbr[s] = (int32_t*)malloc(sizeof(int32_t) * (size_t)sy->N * (size_t)sy->z[s]);
        if (!sy->nbr[s]) return -1;
        for (int64_t a = 0; a < sy->N; a++) {
            int p[3]; site_position(sy, a, p);
            for (int k = 0; k < sy->z[s]; k++) {
                int q[3];
                for (int d = 0; d < 3; d++) q[d] = posmod(p[d] + offs[s][k][d], 2*sy->L[d]);   /* periodic */
                int64_t v = site_of_position(sy, q);
                if (v < 0) return -2;
                sy->nbr[s][a*sy->z[s] + k] = (int32_t)v;
            }
        }
    }
    return 0;
}

/* ---------------------------------------------------------------- D3: species counts */
/* N_i = round(c_i N) when c_i N is within 1e-9 of an integer, else floor + largest remainder (ties -> lower index). */
static int species_counts(int64_t N, int M, const double *conc, int64_t *out)
{
    double sum = 0.0, rem[ORA_MAX_SPECIES];
    int64_t tot = 0;
    for (int i = 0; i < M; i++) { if (!(conc[i] > 0.0)) return -1; sum += conc[i]; }
    if (fabs(sum - 1.0) > 1e-9) return -1;
    for (int i = 0; i < M; i++) {
        double x = conc[i] * (double)N;
        double r = floor(x + 0.5);
        if (fabs(x - r) <= 1e-9) { out[i] = (int64_t)r; rem[i] = 0.0; }
        else { out[i] = (int64_t)floor(x); rem[i] = x - floor(x); }
        tot += out[i];
    }
    while (tot < N) {                       /* largest remainder, ties -> lower index */
        int best = 0;
        for (int i = 1; i < M; i++) if (rem[i] > rem[best]) best = i;
        out[best]++; rem[best] = -1.0; tot++;
    }
    if (tot != N) return -1;
    for (int i = 0; i < M; i++) if (out[i] <= 0) return -1;
    return 0;
}

/* ---------------------------------------------------------------- create / destroy / info */
ora_sys *ora_create(int lattice, int Lx, int Ly, int Lz, int M, const double *conc,
                    int S, const double *shell_w, const double *alpha_target)
{
    if (lattice < 0 || lattice > 1 || Lx < 1 || Ly < 1 || Lz < 1) return NULL;
    if (M < 1 || M > ORA_MAX_SPECIES || S < 1 || S > ORA_MAX_SHELLS) return NULL;
    ora_sys *sy = (ora_sys*)calloc(1, sizeof(ora_sys));
    if (!sy) return NULL;
    sy->lattice = lattice; sy->L[0] = Lx; sy->L[1] = Ly; sy->L[2] = Lz;
    sy->A = lattice == 0 ? 4 : 2;
    sy->N = (int64_t)sy->A * Lx * Ly * Lz;
    sy->M = M; sy->S = S;
    if (sy->N >= ((int64_t)1 << 31) || species_counts(sy->N, M, conc, sy->n_per_species) != 0) { free(sy); return NULL; }
    if (build_tables(sy) != 0) { for (int s = 0; s < S; s++) free(sy->nbr[s]); free(sy); return NULL; }
    for (int s = 0; s < S; s++) {
        sy->w[s] = shell_w[s];
        for (int i = 0; i < M; i++) for (int j = 0; j < M; j++) {
            sy->t[s][i][j] = alpha_target[(s*M + i)*M + j];
            /* D6: den exact in fp64 (< 2^53), one correctly rounded divide */
            double den = (double)((int64_t)sy->z[s] * sy->n_per_species[i] * sy->n_per_species[j]);
            sy->g[s][i][j] = (double)sy->N / den;
        }
    }
    return sy;
}

void ora_destroy(ora_sys *sy)
{
    if (!sy) return;
    for (int s = 0; s < ORA_MAX_SHELLS; s++) free(sy->nbr[s]);
    free(sy);
}

void ora_info(const ora_sys *sy, int64_t *n_sites, int *z, int64_t *n_per_species)
{
    *n_sites = sy->N;
    for (int s = 0; s < sy->S; s++) z[s] = sy->z[s];
    for (int i = 0; i < sy->M; i++) n_per_species[i] = sy->n_per_species[i];
}

void ora_neighbor_table(const ora_sys *sy, int shell, int32_t *out)
{
    memcpy(out, sy->nbr[shell], sizeof(int32_t) * (size_t)sy->N * (size_t)sy->z[shell]);
}

/* ---------------------------------------------------------------- D7: Philox4x32-10 */
void ora_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; round++) {
        if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }     /* key bumped between rounds */
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static uint32_t bounded(uint32_t r, uint32_t n) { return (uint32_t)(((uint64_t)r * (uint64_t)n) >> 32); }

/* ---------------------------------------------------------------- D8: Fisher-Yates init */
void ora_init_random(const ora_sys *sy, uint8_t *occ, int64_t C, uint64_t seed, uint64_t chain0)
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    for (int64_t c = 0; c < C; c++) {
        uint8_t *o = occ + c * sy->N;
        int64_t n = 0;
        for (int i = 0; i < sy->M; i++)
            for (int64_t r = 0; r < sy->n_per_species[i]; r++) o[n++] = (uint8_t)i;
        uint32_t chain = (uint32_t)(chain0 + (uint64_t)c);
        for (int64_t m = sy->N - 1; m >= 1; m--) {
            uint32_t ctr[4] = { (uint32_t)m, 0u, 0xFFFFFFFFu, chain }, r[4];
            ora_philox4x32_10(ctr, key, r);
            uint32_t j = bounded(r[0], (uint32_t)(m + 1));
            uint8_t tmp = o[m]; o[m] = o[j]; o[j] = tmp;
        }
    }
}

/* ---------------------------------------------------------------- D4: pair counts (the recount) */
/* counts[s][i][j] = #{(a, k) : occ[a] = i, occ[nbr_s[a][k]] = j}  -- ordered pairs over TABLE ENTRIES */
void ora_pair_counts(const ora_sys *sy, const uint8_t *occ, int32_t *counts)
{
    int M = sy->M;
    memset(counts, 0, sizeof(int32_t) * (size_t)(sy->S * M * M));
    for (int s = 0; s < sy->S; s++)
        for (int64_t a = 0; a < sy->N; a++)
            for (int k = 0; k < sy->z[s]; k++) {
                int i = occ[a], j = occ[sy->nbr[s][a*sy->z[s] + k]];
                counts[(s*M + i)*M + j] += 1;
            }
}

/* ---------------------------------------------------------------- D5: alpha (Eq. 2) */
void ora_alpha(const ora_sys *sy, const int32_t *counts, double *alpha)
{
    int M = sy->M;
    for (int s = 0; s < sy->S; s++) for (int i = 0; i < M; i++) for (int j = 0; j < M; j++) {
        double x = (double)counts[(s*M + i)*M + j] * sy->g[s][i][j];
        alpha[(s*M + i)*M + j] = 1.0 - x;
    }
}

/* ---------------------------------------------------------------- D6: objective J = F^2 (Eq. 3) */
double ora_objective(const ora_sys *sy, const int32_t *counts)
{
    int M = sy->M;
    double J = 0.0;
    for (int s = 0; s < sy->S; s++) {
        double sh = 0.0;
        for (int i = 0; i < M; i++) {
            double row = 0.0;
            for (int j = 0; j < M; j++) {
                double x  = (double)counts[(s*M + i)*M + j] * sy->g[s][i][j];
                double al = 1.0 - x;
                double d  = al - sy->t[s][i][j];
                double e  = d * d;
                row = row + e;
            }
            sh = sh + row;
        }
        J = J + sy->w[s] * sh;
    }
    return J;
}

void ora_sro_full(const ora_sys *sy, const uint8_t *occ, int64_t B, int32_t *counts, double *alpha, double *J)
{
    int sz = sy->S * sy->M * sy->M;
    for (int64_t b = 0; b < B; b++) {
        ora_pair_counts(sy, occ + b*sy->N, counts + b*sz);
        if (alpha) ora_alpha(sy, counts + b*sz, alpha + b*sz);
        if (J) J[b] = ora_objective(sy, counts + b*sz);
    }
}

/* ---------------------------------------------------------------- D9: Monte Carlo step */
/* D9.1: proposal for (step, k, chain).  Returns 1 and (a,b) if a pair of unlike species was drawn, 0 = null. */
int ora_propose(const ora_sys *sy, const uint8_t *occ, uint64_t seed, uint64_t chain, uint64_t step, uint32_t k,
                uint32_t *a_out, uint32_t *b_out)
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { (uint32_t)step, (uint32_t)(step >> 32), k, (uint32_t)chain }, r[4];
    ora_philox4x32_10(ctr, key, r);
    uint32_t N = (uint32_t)sy->N;
    uint32_t a = bounded(r[0], N), b = bounded(r[1], N - 1);
    if (b >= a) b++;
    if (occ[a] == occ[b]) {                 /* one redraw with (r2, r3) */
        a = bounded(r[2], N); b = bounded(r[3], N - 1);
        if (b >= a) b++;
        if (occ[a] == occ[b]) { *a_out = a; *b_out = b; return 0; }
    }
    *a_out = a; *b_out = b;
    return 1;
}

/* D9.2 (Eq. 4): add to `counts` the change of the ordered pair counts when the species on
 * sites a and b (p = occ[a] != q = occ[b]) are exchanged.  occ is the configuration BEFORE the swap. */
void ora_delta_counts(const ora_sys *sy, const uint8_t *occ, uint32_t a, uint32_t b, int32_t *counts)
{
    int M = sy->M;
    int p = occ[a], q = occ[b];
    for (int s = 0; s < sy->S; s++) {
        int32_t *Ns = counts + s*M*M;
        for (int which = 0; which < 2; which++) {
            uint32_t u = which == 0 ? a : b;
            int oldsp = which == 0 ? p : q, newsp = which == 0 ? q : p;
            for (int k = 0; k < sy->z[s]; k++) {
                uint32_t v = (uint32_t)sy->nbr[s][(int64_t)u*sy->z[s] + k];
                if (v == a || v == b) continue;
                int r = occ[v];
                Ns[oldsp*M + r]--; Ns[r*M + oldsp]--;
                Ns[newsp*M + r]++; Ns[r*M + newsp]++;
            }
        }
    }
}

static uint64_t hash_word(uint64_t h, uint32_t word) { return (h ^ (uint64_t)word) * 0x100000001b3ULL; }

/* One chain, n_steps steps.  eval_all != 0: every one of the K candidates is evaluated each step (the timed
 * mode: trial count == C*steps*K); eval_all == 0: stop evaluating J at the first improving k (same trajectory,
 * n_null still counts all K slots because nullness does not depend on J). */
static void mc_chain(const ora_sys *sy, uint8_t *occ, int32_t *counts, uint64_t n_steps, int K, uint64_t seed,
                     uint64_t chain, uint64_t step0, ora_stats *st, ora_move *log, int64_t log_cap, int eval_all)
{
    int sz = sy->S * sy->M * sy->M;
    int32_t trial[ORA_MAX_SHELLS*ORA_MAX_SPECIES*ORA_MAX_SPECIES];
    int32_t chosen[ORA_MAX_SHELLS*ORA_MAX_SPECIES*ORA_MAX_SPECIES];
    double J_cur = ora_objective(sy, counts);
    int64_t n_logged = 0;
    for (uint64_t t = 0; t < n_steps; t++) {
        uint64_t step = step0 + t;
        int found = 0; uint32_t ks = 0, as = 0, bs = 0; double Js = 0.0;
        for (int k = 0; k < K; k++) {
            uint32_t a, b;
            if (!ora_propose(sy, occ, seed, chain, step, (uint32_t)k, &a, &b)) { st->n_null++; continue; }
            if (found && !eval_all) continue;
            memcpy(trial, counts, sizeof(int32_t)*sz);
            ora_delta_counts(sy, occ, a, b, trial);
            double Jk = ora_objective(sy, trial);
            if (!found && Jk < J_cur) {             /* lowest k with strict improvement */
                found = 1; ks = (uint32_t)k; as = a; bs = b; Js = Jk;
                memcpy(chosen, trial, sizeof(int32_t)*sz);
            }
        }
        if (found) {
            uint8_t tmp = occ[as]; occ[as] = occ[bs]; occ[bs] = tmp;
            memcpy(counts, chosen, sizeof(int32_t)*sz);
            J_cur = Js;
            st->n_accept++;
            st->last_accept_step = step;
            uint64_t h = st->hash;
            h = hash_word(h, (uint32_t)step); h = hash_word(h, (uint32_t)(step >> 32));
            h = hash_word(h, ks); h = hash_word(h, as); h = hash_word(h, bs);
            st->hash = h;
            if (log && n_logged < log_cap) { ora_move m = { step, ks, as, bs }; log[n_logged++] = m; }
        }
    }
    st->J = J_cur;
}

/* ---- the paper's own selection and termination, as options (Eq. 6: F_best = min over the
 * candidates; Alg. 3 P:244-250 and section 4.6.4: a search-depth counter, reset when a better solution is
 * found, incremented otherwise, the search ending when it reaches its threshold or after the maximum number of steps).
 * Reading (A23): select_best != 0 -> the candidate with the smallest J_k is taken (ties -> lowest k) and
 * applied iff J_k < J_cur (tolerance 0, as in D9); depth = consecutive steps without an applied move; with
 * depth_limit > 0 a chain stops as soon as depth == depth_limit (a chain entering with depth >= depth_limit does nothing).
 * depth is in/out so that split runs continue exactly; *steps_done = steps executed by this call.
 * Every K candidates are evaluated in best mode (the minimum needs all of them). */
static void mc_chain_ex(const ora_sys *sy, uint8_t *occ, int32_t *counts, uint64_t n_steps, int K, uint64_t seed,
                        uint64_t chain, uint64_t step0, ora_stats *st, ora_move *log, int64_t log_cap,
                        int select_best, uint64_t depth_limit, uint64_t *depth_io, uint64_t *steps_done)
{
    int sz = sy->S * sy->M * sy->M;
    int32_t trial[ORA_MAX_SHELLS*ORA_MAX_SPECIES*ORA_MAX_SPECIES];
    int32_t chosen[ORA_MAX_SHELLS*ORA_MAX_SPECIES*ORA_MAX_SPECIES];
    double J_cur = ora_objective(sy, counts);
    int64_t n_logged = 0;
    uint64_t depth = depth_io ? *depth_io : 0;
    uint64_t t = 0;
    for (; t < n_steps; t++) {
        if (depth_limit > 0 && depth >= depth_limit) break;
        uint64_t step = step0 + t;
        int found = 0; uint32_t ks = 0, as = 0, bs = 0; double Js = 0.0;
        for (int k = 0; k < K; k++) {
            uint32_t a, b;
            if (!ora_propose(sy, occ, seed, chain, step, (uint32_t)k, &a, &b)) { st->n_null++; continue; }
            if (found && !select_best) continue;
            memcpy(trial, counts, sizeof(int32_t)*sz);
            ora_delta_counts(sy, occ, a, b, trial);
            double Jk = ora_objective(sy, trial);
            int take = select_best ? (Jk < J_cur && (!found || Jk < Js))      /* strict: ties keep the lower k */
                                   : (!found && Jk < J_cur);
            if (take) {
                found = 1; ks = (uint32_t)k; as = a; bs = b; Js = Jk;
                memcpy(chosen, trial, sizeof(int32_t)*sz);
            }
        }
        if (found) {
            uint8_t tmp = occ[as]; occ[as] = occ[bs]; occ[bs] = tmp;
            memcpy(counts, chosen, sizeof(int32_t)*sz);
            J_cur = Js;
            st->n_accept++;
            st->last_accept_step = step;
            uint64_t h = st->hash;
            h = hash_word(h, (uint32_t)step); h = hash_word(h, (uint32_t)(step >> 32));
            h = hash_word(h, ks); h = hash_word(h, as); h = hash_word(h, bs);
            st->hash = h;
            if (log && n_logged < log_cap) { ora_move m = { step, ks, as, bs }; log[n_logged++] = m; }
            depth = 0;
        } else {
            depth++;
        }
    }
    st->J = J_cur;
    if (depth_io) *depth_io = depth;
    if (steps_done) *steps_done = t;
}

/* single-threaded over the chains (a test oracle, not the timed baseline) */
int ora_mc_run_ex(const ora_sys *sy, uint8_t *occ, int32_t *counts, int64_t C, uint64_t n_steps, int K,
                  uint64_t seed, uint64_t chain0, uint64_t step0, ora_stats *stats, ora_move *log, int64_t log_cap,
                  int select_best, uint64_t depth_limit, uint64_t *depth_io, uint64_t *steps_done)
{
    int sz = sy->S * sy->M * sy->M;
    for (int64_t c = 0; c < C; c++)
        mc_chain_ex(sy, occ + c*sy->N, counts + c*sz, n_steps, K, seed, chain0 + (uint64_t)c, step0, stats + c,
                    log ? log + c*log_cap : NULL, log_cap, select_best, depth_limit,
                    depth_io ? depth_io + c : NULL, steps_done ? steps_done + c : NULL);
    return 1;
}

typedef struct {
    const ora_sys *sy; uint8_t *occ; int32_t *counts; int64_t c_begin, c_end; uint64_t n_steps; int K;
    uint64_t seed, chain0, step0; ora_stats *stats; ora_move *log; int64_t log_cap; int eval_all;
} mc_job;

static void *mc_worker(void *arg)
{
    mc_job *j = (mc_job*)arg;
    int sz = j->sy->S * j->sy->M * j->sy->M;
    for (int64_t c = j->c_begin; c < j->c_end; c++)
        mc_chain(j->sy, j->occ + c*j->sy->N, j->counts + c*sz, j->n_steps, j->K, j->seed, j->chain0 + (uint64_t)c,
                 j->step0, j->stats + c, j->log ? j->log + c*j->log_cap : NULL, j->log_cap, j->eval_all);
    return NULL;
}

/* stats[c] is in/out: n_accept, n_null, hash, last_accept_step continue; J is overwritten.
 * Initial stats for a fresh chain: {0, 0, 0xcbf29ce484222325, UINT64_MAX, 0}.  Returns the threads used. */
int ora_mc_run(const ora_sys *sy, uint8_t *occ, int32_t *counts, int64_t C, uint64_t n_steps, int K,
               uint64_t seed, uint64_t chain0, uint64_t step0, ora_stats *stats, ora_move *log, int64_t log_cap,
               int n_threads, int eval_all)
{
    if (n_threads < 1) n_threads = 1;
    if (n_threads > C) n_threads = (int)(C > 0 ? C : 1);
    if (n_threads > 256) n_threads = 256;
    pthread_t th[256]; mc_job jobs[256];
    for (int t = 0; t < n_threads; t++) {
        mc_job j = { sy, occ, counts, C * t / n_threads, C * (t + 1) / n_threads, n_steps, K, seed, chain0, step0,
                     stats, log, log_cap, eval_all };
        jobs[t] = j;
    }
    if (n_threads == 1) { mc_worker(&jobs[0]); return 1; }
    for (int t = 0; t < n_threads; t++) pthread_create(&th[t], NULL, mc_worker, &jobs[t]);
    for (int t = 0; t < n_threads; t++) pthread_join(th[t], NULL);
    return n_threads;
}

/* threaded recount over the batch (timed baseline for hea_sro_full); returns the threads used */
typedef struct { const ora_sys *sy; const uint8_t *occ; int64_t b0, b1; int32_t *counts; double *alpha; double *J; } sro_job;
static void *sro_worker(void *arg)
{
    sro_job *j = (sro_job*)arg;
    int sz = j->sy->S * j->sy->M * j->sy->M;
    if (j->b1 > j->b0)
        ora_sro_full(j->sy, j->occ + j->b0*j->sy->N, j->b1 - j->b0, j->counts + j->b0*sz,
                     j->alpha ? j->alpha + j->b0*sz : NULL, j->J ? j->J + j->b0 : NULL);
    return NULL;
}
int ora_sro_full_mt(const ora_sys *sy, const uint8_t *occ, int64_t B, int32_t *counts, double *alpha, double *J,
                    int n_threads)
{
    if (n_threads < 1) n_threads = 1;
    if (n_threads > B) n_threads = (int)(B > 0 ? B : 1);
    if (n_threads > 256) n_threads = 256;
    pthread_t th[256]; sro_job jobs[256];
    for (int t = 0; t < n_threads; t++) {
        sro_job j = { sy, occ, B * t / n_threads, B * (t + 1) / n_threads, counts, alpha, J };
        jobs[t] = j;
    }
    if (n_threads == 1) { sro_worker(&jobs[0]); return 1; }
    for (int t = 0; t < n_threads; t++) pthread_create(&th[t], NULL, sro_worker, &jobs[t]);
    for (int t = 0; t < n_threads; t++) pthread_join(th[t], NULL);
    return n_threads;
}
