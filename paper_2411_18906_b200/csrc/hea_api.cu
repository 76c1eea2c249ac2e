// hea_api.cu -- the C ABI of libhea_b200 (include/hea.h): context, validation, launches.  No torch types.
#include "../../include/hea.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "hea_device.cuh"
#include "hea_lattice.hpp"

namespace hea {
// launchers (hea_sro.cu / hea_mc.cu)
cudaError_t launch_sro_count(const KParams& P, int lat, const uint8_t* occ, int64_t B, int32_t* counts, int n_sms,
                             size_t smem_budget, int opt_stages, int opt_blocks_per_sm, int opt_warps, cudaStream_t st, int64_t* n_launches);
bool sro_stencil_usable(const Lattice& lat, const uint8_t* occ);
cudaError_t launch_sro_stencil(const KParams& P, const Lattice& lat, const uint8_t* occ, int64_t B, int32_t* counts,
                               int n_sms, int tile_xy, int tile_z, int blocks_per_sm, int flush_tiles, int opt_threads,
                               int lanes, cudaStream_t st,
                               int64_t* n_launches);
cudaError_t launch_sro_epilogue(const KParams& P, const int32_t* counts, int64_t B, double* alpha, double* obj,
                                cudaStream_t st, int64_t* n_launches);
cudaError_t launch_init_random(const KParams& P, uint8_t* occ, int64_t C, uint64_t seed, uint64_t chain0,
                               const int64_t* n_per_species_dev, size_t smem_budget, cudaStream_t st, int64_t* n_launches);
cudaError_t launch_stats_reset(void* stats, int64_t C, cudaStream_t st, int64_t* n_launches);
size_t mc_shared_bytes(int occ_mode, int N, int AZ, bool fast_nbr);
cudaError_t launch_mc(const KParams& P, const DevTables& host_tab, int occ_mode, int threads, int cluster, int w_max,
                      bool fast_nbr, uint8_t* occ, int32_t* counts, int64_t C, uint64_t n_steps, int K, uint64_t seed, uint64_t chain0,
                      uint64_t step0, void* stats, void* log, int64_t log_cap, cudaStream_t st, int64_t* n_launches,
                      int* query_max_clusters);
size_t mc2_shared_bytes(int occ_mode, int lattice, const int* L, int M);
cudaError_t launch_pool_rank(const double* J, int64_t C, int64_t n_keep, int32_t* order, cudaStream_t st, int64_t* n_launches);
cudaError_t launch_pool_gather(const void* src, void* dst, const int32_t* order, int64_t n_keep, size_t item,
                               cudaStream_t st, int64_t* n_launches);
size_t mc2_team_bytes(int64_t C);
cudaError_t measure_peaks(int n_sms, int clock_khz, double* out, cudaStream_t st, int64_t* n_launches);
cudaError_t pool_rank_static(const KParams& P, int device, const int32_t* counts, int64_t C, int64_t n_keep, int32_t* order,
                             cudaStream_t st, int64_t* n_launches, std::string* err);
constexpr int kMc2MaxThreads = 512;
cudaError_t launch_mc2(const KParams& P, const DevTables& host_tab, int lattice, int occ_mode, int threads, int team,
                       void* team_ctl, int team_on, int team_off, int accept_engine, size_t smem_budget, int w_max, uint8_t* occ, int32_t* counts, int64_t C, uint64_t n_steps, int K, uint64_t seed, uint64_t chain0,
                       uint64_t step0, void* stats, void* log, int64_t log_cap, int select_best, uint64_t depth_limit,
                       uint64_t* depth, uint64_t* steps_done, uint32_t* hist, cudaStream_t st, int64_t* n_launches);
}  // namespace hea

struct hea_ctx {
    hea::Lattice lat;
    int M = 0, S = 0;
    int64_t n_per_species[hea::kMaxSpecies] = {0};
    int device = 0;
    int n_sms = 0;
    size_t smem_optin = 0;
    int32_t* d_nbr_site = nullptr;
    hea::DevTables* d_tab = nullptr;
    hea::DevTables tab_host{};
    int64_t* d_nps = nullptr;
    hea::KParams P{};
    // tuning options (0 = auto)
    int64_t opt_occ_mode = 0, opt_threads = 0, opt_cluster = 0, opt_window = 0, opt_neighbors = 0, opt_engine = 0, opt_team = 0, opt_team_on = 0, opt_team_off = 0, opt_accept = 0, opt_hist = 0, opt_sro_stages = 0, opt_sro_bps = 0, opt_sro_warps = 0, opt_sro_engine = 0, opt_sro_tile_xy = 0, opt_sro_tile_z = 0, opt_sro_flush = 0, opt_sro_threads = 0, opt_sro_lanes = 0;
    int64_t n_launches = 0;
    // internal stream and scratch for the *_host entry points
    cudaStream_t stream = nullptr;
    void* scratch[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    size_t scratch_cap[7] = {0, 0, 0, 0, 0, 0, 0};
};

namespace {

thread_local std::string g_err = "";

int fail(int code, const std::string& msg)
{
    g_err = msg;
    return code;
}

int fail_cuda(cudaError_t e, const char* what)
{
    g_err = std::string(what) + ": " + cudaGetErrorString(e);
    return HEA_ECUDA;
}

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; prev = -1; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

int ensure_scratch(hea_ctx* ctx, int slot, size_t bytes)
{
    if (ctx->scratch_cap[slot] >= bytes) return HEA_OK;
    if (ctx->scratch[slot]) cudaFree(ctx->scratch[slot]);
    ctx->scratch[slot] = nullptr;
    ctx->scratch_cap[slot] = 0;
    cudaError_t e = cudaMalloc(&ctx->scratch[slot], bytes);
    if (e != cudaSuccess) return fail(HEA_ENOMEM, std::string("cudaMalloc scratch: ") + cudaGetErrorString(e));
    ctx->scratch_cap[slot] = bytes;
    return HEA_OK;
}

int64_t* option_slot(hea_ctx* ctx, const char* name)
{
    if (!name) return nullptr;
    if (!strcmp(name, "mc_occ_mode")) return &ctx->opt_occ_mode;
    if (!strcmp(name, "mc_threads")) return &ctx->opt_threads;
    if (!strcmp(name, "mc_cluster")) return &ctx->opt_cluster;
    if (!strcmp(name, "mc_window")) return &ctx->opt_window;
    if (!strcmp(name, "mc_neighbors")) return &ctx->opt_neighbors;
    if (!strcmp(name, "mc_engine")) return &ctx->opt_engine;
    if (!strcmp(name, "mc_team")) return &ctx->opt_team;
    if (!strcmp(name, "mc_accept")) return &ctx->opt_accept;
    if (!strcmp(name, "mc_hist")) return &ctx->opt_hist;
    if (!strcmp(name, "mc_team_on")) return &ctx->opt_team_on;
    if (!strcmp(name, "mc_team_off")) return &ctx->opt_team_off;
    if (!strcmp(name, "sro_stages")) return &ctx->opt_sro_stages;
    if (!strcmp(name, "sro_blocks_per_sm")) return &ctx->opt_sro_bps;
    if (!strcmp(name, "sro_warps")) return &ctx->opt_sro_warps;
    if (!strcmp(name, "sro_engine")) return &ctx->opt_sro_engine;
    if (!strcmp(name, "sro_tile_xy")) return &ctx->opt_sro_tile_xy;
    if (!strcmp(name, "sro_tile_z")) return &ctx->opt_sro_tile_z;
    if (!strcmp(name, "sro_flush_tiles")) return &ctx->opt_sro_flush;
    if (!strcmp(name, "sro_threads")) return &ctx->opt_sro_threads;
    if (!strcmp(name, "sro_lanes")) return &ctx->opt_sro_lanes;
    return nullptr;
}

bool option_value_ok(const char* name, int64_t v)
{
    if (v == 0) return true;
    if (!strcmp(name, "mc_occ_mode")) return v >= 1 && v <= 3;
    if (!strcmp(name, "mc_threads")) return v >= 32 && v <= 1024 && v % 32 == 0;
    if (!strcmp(name, "mc_cluster")) return v >= 1 && v <= 8;
    if (!strcmp(name, "mc_window")) return v >= 1 && v <= (1 << 20);
    if (!strcmp(name, "mc_neighbors")) return v == 1 || v == 2;
    if (!strcmp(name, "mc_engine")) return v == 1 || v == 2;
    if (!strcmp(name, "mc_team")) return v >= 1 && v <= 32;
    if (!strcmp(name, "mc_accept")) return v >= 1 && v <= 3;      // 1 off, 2 single-step engine, 3 (= default) pipelined
    if (!strcmp(name, "mc_hist")) return v == 1 || v == 2;        // 1 off, 2 on wherever the kernel can use it
    if (!strcmp(name, "mc_team_on") || !strcmp(name, "mc_team_off")) return v >= 1 && v <= (1 << 30);
    if (!strcmp(name, "sro_stages")) return v >= 1 && v <= 8;
    if (!strcmp(name, "sro_blocks_per_sm")) return v >= 1 && v <= 4;
    if (!strcmp(name, "sro_warps")) return v >= 1 && v <= 16;
    if (!strcmp(name, "sro_engine")) return v == 1 || v == 2;
    if (!strcmp(name, "sro_tile_xy")) return v >= 1 && v <= 8;
    if (!strcmp(name, "sro_tile_z")) return v == 12 || v == 22 || v == 34;
    if (!strcmp(name, "sro_flush_tiles")) return v >= 1 && v <= (1 << 20);
    if (!strcmp(name, "sro_threads")) return v >= 128 && v <= 384 && v % 32 == 0;
    if (!strcmp(name, "sro_lanes")) return v == 1 || v == 2;
    return false;
}

int floor_pow2(int64_t v)
{
    int p = 1;
    while ((int64_t)p * 2 <= v) p *= 2;
    return p;
}

}  // namespace

extern "C" {

const char* hea_version(void) { return "hea-b200 0.1 (sm_100a)"; }

const char* hea_last_error(void) { return g_err.c_str(); }

int hea_create(hea_ctx** out, int lattice, int Lx, int Ly, int Lz, int n_species, const double* conc, int n_shells,
               const double* shell_w, const double* alpha_target, int device)
{
    if (!out) return fail(HEA_EINVAL, "out is NULL");
    *out = nullptr;
    if (!conc || !shell_w || !alpha_target) return fail(HEA_EINVAL, "conc / shell_w / alpha_target is NULL");
    if (n_species < 1 || n_species > HEA_MAX_SPECIES) return fail(HEA_EUNSUPPORTED, "n_species must be in [1, 8]");
    if (n_shells < 1 || n_shells > HEA_MAX_SHELLS) return fail(HEA_EUNSUPPORTED, "n_shells must be in [1, 3]");
    if (lattice != HEA_FCC && lattice != HEA_BCC) return fail(HEA_EINVAL, "lattice must be HEA_FCC or HEA_BCC");

    hea_ctx* ctx = new (std::nothrow) hea_ctx();
    if (!ctx) return fail(HEA_ENOMEM, "out of host memory");
    std::string err = hea::lattice_init(ctx->lat, lattice, Lx, Ly, Lz, n_shells);
    if (!err.empty()) { delete ctx; return fail(HEA_EINVAL, err); }
    {
        // the ordered pair counts (and the packed accumulators of the recount kernels) are int32: N_ij^s <= z_s * N
        int z_max = 0;
        for (int s = 0; s < n_shells; ++s) z_max = std::max(z_max, ctx->lat.z[s]);
        if ((int64_t)z_max * ctx->lat.N >= (1ll << 31)) {
            delete ctx;
            return fail(HEA_EUNSUPPORTED, "max_s(z_s) * N must be < 2^31 (pair counts are int32)");
        }
    }
    for (int s = 0; s < n_shells; ++s)
        if (!std::isfinite(shell_w[s])) { delete ctx; return fail(HEA_EINVAL, "shell weights must be finite"); }
    for (int i = 0; i < n_shells * n_species * n_species; ++i)
        if (!std::isfinite(alpha_target[i])) { delete ctx; return fail(HEA_EINVAL, "alpha_target must be finite"); }
    ctx->M = n_species;
    ctx->S = n_shells;
    err = hea::species_counts(ctx->lat.N, n_species, conc, ctx->n_per_species);
    if (!err.empty()) { delete ctx; return fail(HEA_EINVAL, err); }

    int n_dev = 0;
    cudaError_t e = cudaGetDeviceCount(&n_dev);
    if (e != cudaSuccess || n_dev <= 0) {
        delete ctx;
        return fail(HEA_ECUDA, std::string("no CUDA device available (this library has no CPU fallback): ") +
                                   cudaGetErrorString(e));
    }
    if (device < 0 || device >= n_dev) { delete ctx; return fail(HEA_EINVAL, "device ordinal out of range"); }
    ctx->device = device;
    DeviceGuard guard(device);
    if (!guard.ok) { delete ctx; return fail(HEA_ECUDA, "cudaSetDevice failed"); }
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) { delete ctx; return fail_cuda(e, "cudaGetDeviceProperties"); }
    ctx->n_sms = prop.multiProcessorCount;
    ctx->smem_optin = prop.sharedMemPerBlockOptin;

    const hea::Lattice& lat = ctx->lat;
    const int N = (int)lat.N, Z = lat.Z, M = n_species, S = n_shells;
    const int Npad = (N + 31) & ~31;      // table rows padded to whole 32-site tiles (padding rows point at site 0)

    // constant tables (D5-D6: den exact in fp64, one correctly rounded divide)
    std::vector<hea::DevTables> tab(1);
    memset(tab.data(), 0, sizeof(hea::DevTables));
    for (int s = 0; s < S; ++s) {
        tab[0].w[s] = shell_w[s];
        for (int i = 0; i < M; ++i)
            for (int j = 0; j < M; ++j) {
                const int idx = (s * M + i) * M + j;
                const double den = (double)((int64_t)lat.z[s] * ctx->n_per_species[i] * ctx->n_per_species[j]);
                tab[0].g[idx] = (double)lat.N / den;
                tab[0].t[idx] = alpha_target[idx];
            }
    }
    for (int b = 0; b < lat.A; ++b)
        for (int k = 0; k < Z; ++k) {
            const hea::StencilEntry& st = lat.stencil[b][k];
            int8_t* dst = tab[0].stencil + (b * Z + k) * 4;
            dst[0] = st.nb; dst[1] = st.sx; dst[2] = st.sy; dst[3] = st.sz;
        }

    for (int b = 0; b < lat.A; ++b)
        for (int sh = 0; sh < S; ++sh) {
            int pos = lat.zoff[sh];
            for (int nb = 0; nb < lat.A; ++nb)
                for (int k = lat.zoff[sh]; k < lat.zoff[sh + 1]; ++k)
                    if (lat.stencil[b][k].nb == nb) tab[0].by_basis[b * Z + pos++] = (uint8_t)k;
            // the MC kernel shifts four gathered nibbles at once: every aligned group of four must have one parity of nb
            for (int i = lat.zoff[sh]; i < lat.zoff[sh + 1]; ++i) {
                const int first = lat.zoff[sh] + ((i - lat.zoff[sh]) & ~3);
                if ((lat.stencil[b][tab[0].by_basis[b * Z + i]].nb & 1) != (lat.stencil[b][tab[0].by_basis[b * Z + first]].nb & 1)) {
                    delete ctx;
                    return fail(HEA_EUNSUPPORTED, "internal: shell entries do not group by basis parity");
                }
            }
        }

    auto bail = [&](int code, const std::string& msg) {
        hea_destroy(ctx);
        return fail(code, msg);
    };
    if ((e = cudaStreamCreateWithFlags(&ctx->stream, cudaStreamNonBlocking)) != cudaSuccess)
        return bail(HEA_ECUDA, std::string("cudaStreamCreate: ") + cudaGetErrorString(e));
    if ((e = cudaMalloc(&ctx->d_tab, sizeof(hea::DevTables))) != cudaSuccess ||
        (e = cudaMalloc(&ctx->d_nps, sizeof(int64_t) * hea::kMaxSpecies)) != cudaSuccess ||
        (e = cudaMalloc(&ctx->d_nbr_site, sizeof(int32_t) * (size_t)Npad * Z)) != cudaSuccess)
        return bail(HEA_ENOMEM, std::string("cudaMalloc tables: ") + cudaGetErrorString(e));
    if ((e = cudaMemcpy(ctx->d_tab, tab.data(), sizeof(hea::DevTables), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMemcpy(ctx->d_nps, ctx->n_per_species, sizeof(int64_t) * hea::kMaxSpecies, cudaMemcpyHostToDevice)) != cudaSuccess)
        return bail(HEA_ECUDA, std::string("cudaMemcpy tables: ") + cudaGetErrorString(e));

    // host table builder -> site-major device table, in chunks
    {
        const int64_t chunk_sites = 1 << 20;
        std::vector<int32_t> buf((size_t)std::min<int64_t>(chunk_sites, N) * Z);
        for (int64_t first = 0; first < N; first += chunk_sites) {
            const int64_t last = std::min<int64_t>(N, first + chunk_sites);
            hea::build_site_major(lat, first, last, buf.data());
            e = cudaMemcpy(ctx->d_nbr_site + (size_t)first * Z, buf.data(), sizeof(int32_t) * (size_t)(last - first) * Z,
                           cudaMemcpyHostToDevice);
            if (e != cudaSuccess) return bail(HEA_ECUDA, std::string("cudaMemcpy table: ") + cudaGetErrorString(e));
        }
        if (Npad > N) {
            e = cudaMemset(ctx->d_nbr_site + (size_t)N * Z, 0, sizeof(int32_t) * (size_t)(Npad - N) * Z);
            if (e != cudaSuccess) return bail(HEA_ECUDA, std::string("cudaMemset table padding: ") + cudaGetErrorString(e));
        }
    }

    hea::KParams& P = ctx->P;
    P.N = N; P.Npad = Npad; P.M = M; P.S = S; P.Z = Z; P.A = lat.A;
    for (int d = 0; d < 3; ++d) P.L[d] = lat.L[d];
    for (int s = 0; s < 3; ++s) P.z[s] = s < S ? lat.z[s] : 0;
    for (int s = 0; s < 4; ++s) P.zoff[s] = s <= S ? lat.zoff[s] : Z;
    for (int sh = 0; sh < 3; ++sh) {
        P.m_self[sh] = 0;
        if (sh < S)
            for (int k = lat.zoff[sh]; k < lat.zoff[sh + 1]; ++k) {
                const hea::StencilEntry& st = lat.stencil[0][k];
                if (st.nb == 0 && st.sx % lat.L[0] == 0 && st.sy % lat.L[1] == 0 && st.sz % lat.L[2] == 0) ++P.m_self[sh];
            }
    }
    P.nbr_site = ctx->d_nbr_site;
    P.tab = ctx->d_tab;
    ctx->tab_host = tab[0];
    *out = ctx;
    return HEA_OK;
}

int hea_destroy(hea_ctx* ctx)
{
    if (!ctx) return HEA_OK;
    {
        DeviceGuard guard(ctx->device);
        if (ctx->stream) { cudaStreamSynchronize(ctx->stream); cudaStreamDestroy(ctx->stream); }
        cudaFree(ctx->d_tab);
        cudaFree(ctx->d_nps);
        cudaFree(ctx->d_nbr_site);
        for (void* p : ctx->scratch) cudaFree(p);
    }
    delete ctx;
    return HEA_OK;
}

int hea_info(const hea_ctx* ctx, int64_t* n_sites, int* z, int64_t* n_per_species)
{
    if (!ctx) return fail(HEA_EINVAL, "ctx is NULL");
    if (n_sites) *n_sites = ctx->lat.N;
    if (z) for (int s = 0; s < ctx->S; ++s) z[s] = ctx->lat.z[s];
    if (n_per_species) for (int i = 0; i < ctx->M; ++i) n_per_species[i] = ctx->n_per_species[i];
    return HEA_OK;
}

int hea_neighbor_table(const hea_ctx* ctx, int shell, int32_t* out_host)
{
    if (!ctx || !out_host) return fail(HEA_EINVAL, "ctx / out_host is NULL");
    if (shell < 0 || shell >= ctx->S) return fail(HEA_EINVAL, "shell out of range");
    hea::build_shell_table(ctx->lat, shell, out_host);
    return HEA_OK;
}

int hea_set_option(hea_ctx* ctx, const char* name, int64_t value)
{
    if (!ctx) return fail(HEA_EINVAL, "ctx is NULL");
    int64_t* slot = option_slot(ctx, name);
    if (!slot) return fail(HEA_EINVAL, "unknown option name");
    if (!option_value_ok(name, value)) return fail(HEA_EINVAL, "option value not allowed");
    *slot = value;
    return HEA_OK;
}

int hea_get_option(const hea_ctx* ctx, const char* name, int64_t* value)
{
    if (!ctx || !value) return fail(HEA_EINVAL, "ctx / value is NULL");
    int64_t* slot = option_slot(const_cast<hea_ctx*>(ctx), name);
    if (!slot) return fail(HEA_EINVAL, "unknown option name");
    *value = *slot;
    return HEA_OK;
}

int hea_launch_count(const hea_ctx* ctx, int64_t* n)
{
    if (!ctx || !n) return fail(HEA_EINVAL, "ctx / n is NULL");
    *n = ctx->n_launches;
    return HEA_OK;
}

int hea_init_random(hea_ctx* ctx, uint8_t* occ_dev, int64_t C, uint64_t seed, uint64_t chain0, void* cuda_stream)
{
    if (!ctx) return fail(HEA_EINVAL, "ctx is NULL");
    if (C < 0 || chain0 + (uint64_t)C > (1ull << 32)) return fail(HEA_EINVAL, "chain ids must be < 2^32");
    if (C == 0) return HEA_OK;
    if (!occ_dev) return fail(HEA_EINVAL, "occ_dev is NULL");
    DeviceGuard guard(ctx->device);
    cudaError_t e = hea::launch_init_random(ctx->P, occ_dev, C, seed, chain0, ctx->d_nps, ctx->smem_optin, (cudaStream_t)cuda_stream,
                                            &ctx->n_launches);
    return e == cudaSuccess ? HEA_OK : fail_cuda(e, "hea_init_random launch");
}

int hea_sro_full(hea_ctx* ctx, const uint8_t* occ_dev, int64_t B, int32_t* counts_dev, double* alpha_dev,
                 double* obj_dev, void* cuda_stream)
{
    if (!ctx) return fail(HEA_EINVAL, "ctx is NULL");
    if (B < 0) return fail(HEA_EINVAL, "B must be >= 0");
    if (B == 0) return HEA_OK;                      // empty batch: nothing is read or written, pointers may be NULL
    if (!occ_dev || !counts_dev) return fail(HEA_EINVAL, "occ_dev / counts_dev is NULL");
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // engine: the table-free stencil kernel unless the table-driven one is asked for (or occ is not A-aligned)
    const bool usable = hea::sro_stencil_usable(ctx->lat, occ_dev);
    if (ctx->opt_sro_engine == 2 && !usable) return fail(HEA_EINVAL, "sro_engine 2 needs occ_dev aligned to the basis size");
    cudaError_t e;
    if (ctx->opt_sro_engine != 1 && usable)
        e = hea::launch_sro_stencil(ctx->P, ctx->lat, occ_dev, B, counts_dev, ctx->n_sms, (int)ctx->opt_sro_tile_xy,
                                    (int)ctx->opt_sro_tile_z, (int)ctx->opt_sro_bps, (int)ctx->opt_sro_flush, (int)ctx->opt_sro_threads, (int)ctx->opt_sro_lanes, st, &ctx->n_launches);
    else
        e = hea::launch_sro_count(ctx->P, ctx->lat.type, occ_dev, B, counts_dev, ctx->n_sms, ctx->smem_optin,
                                  (int)ctx->opt_sro_stages, (int)ctx->opt_sro_bps, (int)ctx->opt_sro_warps, st, &ctx->n_launches);
    if (e != cudaSuccess) return fail_cuda(e, "hea_sro_full count launch");
    e = hea::launch_sro_epilogue(ctx->P, counts_dev, B, alpha_dev, obj_dev, st, &ctx->n_launches);
    return e == cudaSuccess ? HEA_OK : fail_cuda(e, "hea_sro_full epilogue launch");
}

int hea_mc_stats_reset(hea_ctx* ctx, hea_mc_stats* stats_dev, int64_t C, void* cuda_stream)
{
    if (!ctx) return fail(HEA_EINVAL, "ctx is NULL");
    if (C < 0) return fail(HEA_EINVAL, "C must be >= 0");
    if (C == 0) return HEA_OK;
    if (!stats_dev) return fail(HEA_EINVAL, "stats_dev is NULL");
    DeviceGuard guard(ctx->device);
    cudaError_t e = hea::launch_stats_reset(stats_dev, C, (cudaStream_t)cuda_stream, &ctx->n_launches);
    return e == cudaSuccess ? HEA_OK : fail_cuda(e, "hea_mc_stats_reset launch");
}

int hea_mc_run(hea_ctx* ctx, uint8_t* occ_dev, int32_t* counts_dev, int64_t C, uint64_t n_steps, int K, uint64_t seed,
               uint64_t chain0, uint64_t step0, hea_mc_stats* stats_dev, hea_move* log_dev, int64_t log_cap,
               void* cuda_stream)
{
    return hea_mc_run_ex(ctx, occ_dev, counts_dev, C, n_steps, K, seed, chain0, step0, stats_dev, log_dev, log_cap, 0, 0,
                         nullptr, nullptr, cuda_stream);
}

int hea_mc_run_ex(hea_ctx* ctx, uint8_t* occ_dev, int32_t* counts_dev, int64_t C, uint64_t n_steps, int K, uint64_t seed,
                  uint64_t chain0, uint64_t step0, hea_mc_stats* stats_dev, hea_move* log_dev, int64_t log_cap,
                  int select_best, uint64_t depth_limit, uint64_t* depth_dev, uint64_t* steps_done_dev, void* cuda_stream)
{
    if (depth_limit > 0 && C != 0 && !depth_dev) return fail(HEA_EINVAL, "depth_limit > 0 needs depth_dev");
    const bool ex_mode = select_best != 0 || depth_limit > 0 || steps_done_dev != nullptr;
    static_assert(sizeof(hea_mc_stats) == 40, "hea_mc_stats layout");
    static_assert(sizeof(hea_move) == 24, "hea_move layout");
    if (!ctx) return fail(HEA_EINVAL, "ctx is NULL");
    if (C != 0 && (!occ_dev || !counts_dev || !stats_dev)) return fail(HEA_EINVAL, "occ_dev / counts_dev / stats_dev is NULL");
    if (K < 1 || K > HEA_MAX_K) return fail(HEA_EINVAL, "K must be in [1, 1024]");
    if (C < 0 || chain0 + (uint64_t)C > (1ull << 32)) return fail(HEA_EINVAL, "chain ids must be < 2^32");
    if (log_cap < 0 || (log_cap > 0 && !log_dev)) return fail(HEA_EINVAL, "log_cap > 0 needs log_dev");
    if (step0 + n_steps < step0) return fail(HEA_EINVAL, "step0 + n_steps overflows");
    if (C == 0) return HEA_OK;
    DeviceGuard guard(ctx->device);
    const int N = ctx->P.N;

    // ---- launch configuration (results never depend on it)
    int occ_mode = (int)ctx->opt_occ_mode;
    const size_t budget = ctx->smem_optin;
    // engine: 2 = halo engine (hea_mc2.cu) whenever the padded one-hot configuration fits in shared memory and no
    // option specific to the window engine (clusters, table neighbours, global occupancy) is set; else 1 (hea_mc.cu)
    int engine = (int)ctx->opt_engine;
    if (engine == 0) {
        const bool fits = hea::mc2_shared_bytes(1, ctx->lat.type, ctx->P.L, ctx->M) <= budget ||
                          (ctx->M <= 4 && hea::mc2_shared_bytes(2, ctx->lat.type, ctx->P.L, ctx->M) <= budget);
        const bool fits_req = occ_mode == 0 || (occ_mode == 1 && hea::mc2_shared_bytes(1, ctx->lat.type, ctx->P.L, ctx->M) <= budget) ||
                              (occ_mode == 2 && ctx->M <= 4 && hea::mc2_shared_bytes(2, ctx->lat.type, ctx->P.L, ctx->M) <= budget);
        engine = (fits && fits_req && ctx->opt_cluster == 0 && ctx->opt_neighbors == 0) ? 2 : 1;
    }
    if (ex_mode && engine != 2)
        return fail(HEA_EUNSUPPORTED, "hea_mc_run_ex options need the shared-memory (halo) engine: configuration too large or engine forced");
    if (engine == 2) {
        // halo engine (hea_mc2.cu): one block per chain, padded one-hot configuration in shared memory
        int om = occ_mode;
        if (om == 0) om = hea::mc2_shared_bytes(1, ctx->lat.type, ctx->P.L, ctx->M) <= budget ? 1 : 2;
        if (om == 3 || (om == 2 && ctx->M > 4) || hea::mc2_shared_bytes(om, ctx->lat.type, ctx->P.L, ctx->M) > budget)
            return fail(HEA_EINVAL, "mc_engine 2: the padded configuration does not fit in shared memory");
        // blocks per chain: a team of R blocks (synchronised through global memory, cooperative launch) when the
        // chains alone would leave at least half of the SMs idle; one block per SM then
        int team = (int)ctx->opt_team;
        if (team == 0) team = (int)std::max<int64_t>(1, std::min<int64_t>(32, ctx->n_sms / C));
        if (team > 1 && (int64_t)team * C > ctx->n_sms) return fail(HEA_EINVAL, "mc_team: team blocks * chains exceeds the SM count");
        int threads = ctx->opt_threads ? (int)ctx->opt_threads : hea::kMc2MaxThreads;
        if (!ctx->opt_threads && team == 1) {
            const int64_t blocks_per_sm = (C + ctx->n_sms - 1) / ctx->n_sms;
            // 128 registers per thread: 512 threads are resident per SM; measured on c2 (7 blocks per SM) and c3 (2 per
            // SM), blocks of 1024 / blocks_per_sm threads running in waves beat smaller blocks that are all resident
            if (blocks_per_sm > 1) threads = std::max(32, std::min(512, floor_pow2(std::max<int64_t>(1, 1024 / blocks_per_sm))));
        }
        threads = std::min(threads, hea::kMc2MaxThreads);   // the halo kernel is compiled for blocks of at most this size
        void* team_ctl = nullptr;
        if (team > 1) {
            int rc = ensure_scratch(ctx, 5, hea::mc2_team_bytes(C));
            if (rc != HEA_OK) return rc;
            team_ctl = ctx->scratch[5];
        }
        // site-histogram table of the reject filter: 4 bytes per site and chain, read through L2.  Default: on
        // while the tables of all chains stay well inside L2 (64 MB); mc_hist = 2 always, mc_hist = 1 never.
        uint32_t* hist = nullptr;
        const size_t hist_bytes = sizeof(uint32_t) * (size_t)N * (size_t)C;
        if (ctx->M >= 2 && ctx->M <= 5 && ctx->opt_hist != 1 && (hist_bytes <= ((size_t)64 << 20) || ctx->opt_hist == 2)) {
            int rc = ensure_scratch(ctx, 6, hist_bytes);
            if (rc != HEA_OK) return rc;
            hist = (uint32_t*)ctx->scratch[6];
        }
        const int w_max2 = ctx->opt_window ? (int)ctx->opt_window : (1 << 20);
        cudaError_t e2 = hea::launch_mc2(ctx->P, ctx->tab_host, ctx->lat.type, om, threads, team, team_ctl,
                                         (int)ctx->opt_team_on, (int)ctx->opt_team_off,
                                         ctx->opt_accept == 1 ? 0 : ctx->opt_accept == 2 ? 1 : 2, budget, w_max2, occ_dev, counts_dev, C,
                                         n_steps, K, seed, chain0, step0, stats_dev, log_dev, log_cap, select_best,
                                         depth_limit, depth_dev, steps_done_dev, hist, (cudaStream_t)cuda_stream,
                                         &ctx->n_launches);
        return e2 == cudaSuccess ? HEA_OK : fail_cuda(e2, "hea_mc_run launch (halo engine)");
    }
    const int AZ = ctx->P.A * ctx->P.Z;
    const bool fast_nbr = ctx->opt_neighbors != 1;      // interior sites: neighbour = site + offset (no table load)
    if (occ_mode == 0) {
        if (hea::mc_shared_bytes(1, N, AZ, fast_nbr) <= budget) occ_mode = 1;
        else if (hea::mc_shared_bytes(2, N, AZ, fast_nbr) <= budget) occ_mode = 2;
        else occ_mode = 3;
    } else if (hea::mc_shared_bytes(occ_mode, N, AZ, fast_nbr) > budget) {
        return fail(HEA_EINVAL, "mc_occ_mode does not fit in shared memory for this N");
    }
    // blocks per chain: spread few chains over the SMs with thread-block clusters (replicated chain state); the
    // largest cluster size for which all C clusters are resident at once (GPC boundaries limit this: 16 clusters of 8
    // do not fit on the 148 SMs of a B200, 16 of 7 do)
    const int w_max = ctx->opt_window ? (int)ctx->opt_window : (1 << 20);
    auto pick_threads = [&](int cl) {
        if (ctx->opt_threads) return (int)ctx->opt_threads;
        // 64 registers per thread -> 1024 resident threads per SM, shared between the blocks that land on one SM
        const int64_t blocks_per_sm = (C * cl + ctx->n_sms - 1) / ctx->n_sms;
        return std::max(32, std::min(1024, floor_pow2(std::max<int64_t>(1, 1024 / blocks_per_sm))));
    };
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int cluster = (int)ctx->opt_cluster;
    if (cluster == 0) {
        cluster = 1;
        for (int cl = 8; cl >= 2; --cl) {
            if (C * cl > ctx->n_sms) continue;
            int fit = 0;
            cudaError_t q = hea::launch_mc(ctx->P, ctx->tab_host, occ_mode, pick_threads(cl), cl, w_max, fast_nbr, occ_dev,
                                           counts_dev, C, n_steps, K, seed, chain0, step0, stats_dev, log_dev, log_cap, st,
                                           &ctx->n_launches, &fit);
            if (q != cudaSuccess) { (void)cudaGetLastError(); continue; }
            if (fit >= C) { cluster = cl; break; }
        }
    }
    cudaError_t e = hea::launch_mc(ctx->P, ctx->tab_host, occ_mode, pick_threads(cluster), cluster, w_max, fast_nbr, occ_dev,
                                   counts_dev, C, n_steps, K, seed, chain0, step0, stats_dev, log_dev, log_cap, st,
                                   &ctx->n_launches, nullptr);
    return e == cudaSuccess ? HEA_OK : fail_cuda(e, "hea_mc_run launch");
}

int hea_pool_select(hea_ctx* ctx, uint8_t* occ_dev, int32_t* counts_dev, hea_mc_stats* stats_dev, int64_t C, int64_t n_keep,
                    uint64_t seed, uint64_t new_chain0, int32_t* order_dev, void* cuda_stream)
{
    if (!ctx) return fail(HEA_EINVAL, "ctx is NULL");
    if (C < 0 || n_keep < 0 || n_keep > C) return fail(HEA_EINVAL, "need 0 <= n_keep <= C");
    if (C > 65536) return fail(HEA_EUNSUPPORTED, "hea_pool_select ranks at most 65,536 chains");
    if (new_chain0 + (uint64_t)(C - n_keep) > (1ull << 32)) return fail(HEA_EINVAL, "chain ids must be < 2^32");
    if (C == 0) return HEA_OK;
    if (!occ_dev || !counts_dev || !stats_dev) return fail(HEA_EINVAL, "occ_dev / counts_dev / stats_dev is NULL");
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t N = (size_t)ctx->P.N, SMM = (size_t)ctx->S * ctx->M * ctx->M;
    int rc;
    if ((rc = ensure_scratch(ctx, 0, N * (size_t)std::max<int64_t>(n_keep, 1))) != HEA_OK) return rc;
    if ((rc = ensure_scratch(ctx, 1, sizeof(int32_t) * SMM * (size_t)std::max<int64_t>(n_keep, 1))) != HEA_OK) return rc;
    if ((rc = ensure_scratch(ctx, 2, sizeof(double) * (size_t)C)) != HEA_OK) return rc;
    if ((rc = ensure_scratch(ctx, 3, sizeof(int32_t) * (size_t)C)) != HEA_OK) return rc;
    if ((rc = ensure_scratch(ctx, 4, sizeof(hea_mc_stats) * (size_t)std::max<int64_t>(n_keep, 1))) != HEA_OK) return rc;
    double* J = (double*)ctx->scratch[2];
    int32_t* order = (int32_t*)ctx->scratch[3];
    cudaError_t e = hea::launch_sro_epilogue(ctx->P, counts_dev, C, nullptr, J, st, &ctx->n_launches);
    if (e == cudaSuccess) e = hea::launch_pool_rank(J, C, n_keep, order, st, &ctx->n_launches);
    if (e == cudaSuccess) e = hea::launch_pool_gather(occ_dev, ctx->scratch[0], order, n_keep, N, st, &ctx->n_launches);
    if (e == cudaSuccess) e = hea::launch_pool_gather(counts_dev, ctx->scratch[1], order, n_keep, sizeof(int32_t) * SMM, st, &ctx->n_launches);
    if (e == cudaSuccess) e = hea::launch_pool_gather(stats_dev, ctx->scratch[4], order, n_keep, sizeof(hea_mc_stats), st, &ctx->n_launches);
    if (e == cudaSuccess && n_keep > 0) {
        e = cudaMemcpyAsync(occ_dev, ctx->scratch[0], N * (size_t)n_keep, cudaMemcpyDeviceToDevice, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(counts_dev, ctx->scratch[1], sizeof(int32_t) * SMM * (size_t)n_keep, cudaMemcpyDeviceToDevice, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(stats_dev, ctx->scratch[4], sizeof(hea_mc_stats) * (size_t)n_keep, cudaMemcpyDeviceToDevice, st);
        if (e == cudaSuccess && order_dev) e = cudaMemcpyAsync(order_dev, order, sizeof(int32_t) * (size_t)n_keep, cudaMemcpyDeviceToDevice, st);
    }
    if (e != cudaSuccess) return fail_cuda(e, "hea_pool_select");
    const int64_t n_new = C - n_keep;
    if (n_new > 0) {
        if ((rc = hea_init_random(ctx, occ_dev + N * (size_t)n_keep, n_new, seed, new_chain0, cuda_stream)) != HEA_OK) return rc;
        if ((rc = hea_sro_full(ctx, occ_dev + N * (size_t)n_keep, n_new, counts_dev + SMM * (size_t)n_keep, nullptr, nullptr, cuda_stream)) != HEA_OK) return rc;
        if ((rc = hea_mc_stats_reset(ctx, stats_dev + n_keep, n_new, cuda_stream)) != HEA_OK) return rc;
    }
    return HEA_OK;
}

int hea_pool_rank_static(hea_ctx* ctx, const int32_t* counts_dev, int64_t C, int64_t n_keep, int32_t* order_dev, void* cuda_stream)
{
    // allocation-free: no ensure_scratch, no cudaMalloc / cudaFree on this path (the scratch is the static array of hea_noalloc.cu)
    if (!ctx) return fail(HEA_EINVAL, "ctx is NULL");
    if (C < 0 || n_keep < 0 || n_keep > C) return fail(HEA_EINVAL, "need 0 <= n_keep <= C");
    if (C > HEA_POOL_RANK_STATIC_MAX)
        return fail(HEA_EINVAL, "hea_pool_rank_static: C = " + std::to_string(C) + " chains exceed the static scratch of HEA_POOL_RANK_STATIC_MAX = " +
                                    std::to_string(HEA_POOL_RANK_STATIC_MAX) + " (use hea_pool_select, which allocates)");
    if (C == 0 || n_keep == 0) return HEA_OK;
    if (!counts_dev || !order_dev) return fail(HEA_EINVAL, "counts_dev / order_dev is NULL");
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail(HEA_ECUDA, "cannot make the context's device current");
    std::string err;
    cudaError_t e = hea::pool_rank_static(ctx->P, ctx->device, counts_dev, C, n_keep, order_dev, (cudaStream_t)cuda_stream,
                                          &ctx->n_launches, &err);
    if (e != cudaSuccess) return fail(HEA_ECUDA, "hea_pool_rank_static: " + err);
    return HEA_OK;
}

int hea_measure_peaks(hea_ctx* ctx, double* out_host, int n_out, void* cuda_stream)
{
    if (!ctx || !out_host) return fail(HEA_EINVAL, "ctx / out_host is NULL");
    if (n_out < HEA_N_PEAKS) return fail(HEA_EINVAL, "out_host needs HEA_N_PEAKS entries");
    DeviceGuard guard(ctx->device);
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, ctx->device);
    cudaError_t e = hea::measure_peaks(ctx->n_sms, khz, out_host, (cudaStream_t)cuda_stream, &ctx->n_launches);
    return e == cudaSuccess ? HEA_OK : fail_cuda(e, "hea_measure_peaks");
}

int hea_sro_full_host(hea_ctx* ctx, const uint8_t* occ_host, int64_t B, int32_t* counts_host, double* alpha_host,
                      double* obj_host)
{
    if (!ctx || !occ_host || !counts_host) return fail(HEA_EINVAL, "ctx / occ_host / counts_host is NULL");
    if (B < 0) return fail(HEA_EINVAL, "B must be >= 0");
    if (B == 0) return HEA_OK;
    DeviceGuard guard(ctx->device);
    const size_t N = (size_t)ctx->P.N, SMM = (size_t)ctx->S * ctx->M * ctx->M;
    int rc;
    if ((rc = ensure_scratch(ctx, 0, N * B)) != HEA_OK) return rc;
    if ((rc = ensure_scratch(ctx, 1, sizeof(int32_t) * SMM * B)) != HEA_OK) return rc;
    if (alpha_host && (rc = ensure_scratch(ctx, 2, sizeof(double) * SMM * B)) != HEA_OK) return rc;
    if (obj_host && (rc = ensure_scratch(ctx, 3, sizeof(double) * B)) != HEA_OK) return rc;
    cudaStream_t st = ctx->stream;
    cudaError_t e = cudaMemcpyAsync(ctx->scratch[0], occ_host, N * B, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return fail_cuda(e, "H2D occ");
    rc = hea_sro_full(ctx, (const uint8_t*)ctx->scratch[0], B, (int32_t*)ctx->scratch[1],
                      alpha_host ? (double*)ctx->scratch[2] : nullptr, obj_host ? (double*)ctx->scratch[3] : nullptr, st);
    if (rc != HEA_OK) return rc;
    e = cudaMemcpyAsync(counts_host, ctx->scratch[1], sizeof(int32_t) * SMM * B, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && alpha_host)
        e = cudaMemcpyAsync(alpha_host, ctx->scratch[2], sizeof(double) * SMM * B, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && obj_host)
        e = cudaMemcpyAsync(obj_host, ctx->scratch[3], sizeof(double) * B, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return e == cudaSuccess ? HEA_OK : fail_cuda(e, "hea_sro_full_host");
}

int hea_mc_run_host(hea_ctx* ctx, uint8_t* occ_host, int32_t* counts_host, int64_t C, uint64_t n_steps, int K,
                    uint64_t seed, uint64_t chain0, uint64_t step0, hea_mc_stats* stats_host)
{
    if (!ctx || !occ_host || !stats_host) return fail(HEA_EINVAL, "ctx / occ_host / stats_host is NULL");
    if (C < 0) return fail(HEA_EINVAL, "C must be >= 0");
    if (C == 0) return HEA_OK;
    DeviceGuard guard(ctx->device);
    const size_t N = (size_t)ctx->P.N, SMM = (size_t)ctx->S * ctx->M * ctx->M;
    int rc;
    if ((rc = ensure_scratch(ctx, 0, N * C)) != HEA_OK) return rc;
    if ((rc = ensure_scratch(ctx, 1, sizeof(int32_t) * SMM * C)) != HEA_OK) return rc;
    if ((rc = ensure_scratch(ctx, 4, sizeof(hea_mc_stats) * C)) != HEA_OK) return rc;
    cudaStream_t st = ctx->stream;
    cudaError_t e = cudaMemcpyAsync(ctx->scratch[0], occ_host, N * C, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(ctx->scratch[4], stats_host, sizeof(hea_mc_stats) * C, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return fail_cuda(e, "H2D occ/stats");
    rc = hea_sro_full(ctx, (const uint8_t*)ctx->scratch[0], C, (int32_t*)ctx->scratch[1], nullptr, nullptr, st);
    if (rc != HEA_OK) return rc;
    rc = hea_mc_run(ctx, (uint8_t*)ctx->scratch[0], (int32_t*)ctx->scratch[1], C, n_steps, K, seed, chain0, step0,
                    (hea_mc_stats*)ctx->scratch[4], nullptr, 0, st);
    if (rc != HEA_OK) return rc;
    e = cudaMemcpyAsync(occ_host, ctx->scratch[0], N * C, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && counts_host)
        e = cudaMemcpyAsync(counts_host, ctx->scratch[1], sizeof(int32_t) * SMM * C, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(stats_host, ctx->scratch[4], sizeof(hea_mc_stats) * C, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return e == cudaSuccess ? HEA_OK : fail_cuda(e, "hea_mc_run_host");
}

}  // extern "C"
