// hea_lattice.cpp -- see hea_lattice.hpp.  DESIGN.md D1-D3.
#include "hea_lattice.hpp"

#include <algorithm>
#include <array>
#include <cmath>
#include <thread>

namespace hea {

namespace {

struct Vec { int x, y, z; };

// Basis positions in units of a/2 (D1).
const Vec kFcc[4] = {{0, 0, 0}, {0, 1, 1}, {1, 0, 1}, {1, 1, 0}};
const Vec kBcc[2] = {{0, 0, 0}, {1, 1, 1}};

inline const Vec* basis(int type) { return type == 0 ? kFcc : kBcc; }

// Which basis position has the parity pattern of q?  (Box sides 2L are even, so parity survives the wrap.)
inline int basis_by_parity(int type, int A, const Vec& q)
{
    const Vec* bs = basis(type);
    for (int b = 0; b < A; ++b)
        if (((q.x - bs[b].x) & 1) == 0 && ((q.y - bs[b].y) & 1) == 0 && ((q.z - bs[b].z) & 1) == 0) return b;
    return -1;
}

inline int wrap(int v, int L)
{
    v %= L;
    return v < 0 ? v + L : v;
}

}  // namespace

std::string lattice_init(Lattice& lat, int type, int Lx, int Ly, int Lz, int n_shells)
{
    if (type != 0 && type != 1) return "lattice must be HEA_FCC or HEA_BCC";
    if (Lx < 1 || Ly < 1 || Lz < 1) return "supercell dimensions must be >= 1";
    if (n_shells < 1 || n_shells > kMaxShells) return "n_shells must be in [1, 3]";
    lat.type = type;
    lat.L[0] = Lx; lat.L[1] = Ly; lat.L[2] = Lz;
    lat.A = type == 0 ? 4 : 2;
    const int64_t n = (int64_t)lat.A * Lx * Ly * Lz;
    if (n >= (int64_t(1) << 31)) return "too many sites (N must be < 2^31)";
    lat.N = n;
    lat.S = n_shells;

    // Bravais-lattice vectors from the origin site = differences to every basis position in nearby cells.
    // Collect (|o|^2, o) for all translations within +-2 cells, sort by length then lexicographically (D2).
    std::vector<std::array<int, 4>> vecs;
    const Vec* bs = basis(type);
    for (int cx = -2; cx <= 2; ++cx)
        for (int cy = -2; cy <= 2; ++cy)
            for (int cz = -2; cz <= 2; ++cz)
                for (int b = 0; b < lat.A; ++b) {
                    const int ox = 2 * cx + bs[b].x, oy = 2 * cy + bs[b].y, oz = 2 * cz + bs[b].z;
                    const int d2 = ox * ox + oy * oy + oz * oz;
                    if (d2 > 0) vecs.push_back({d2, ox, oy, oz});
                }
    std::sort(vecs.begin(), vecs.end());
    vecs.erase(std::unique(vecs.begin(), vecs.end()), vecs.end());

    std::vector<std::array<int, 3>> offs;
    size_t pos = 0;
    lat.zoff[0] = 0;
    for (int s = 0; s < n_shells; ++s) {
        const int d2 = vecs[pos][0];
        int zs = 0;
        while (pos < vecs.size() && vecs[pos][0] == d2) {
            offs.push_back({vecs[pos][1], vecs[pos][2], vecs[pos][3]});
            ++pos; ++zs;
        }
        lat.z[s] = zs;
        lat.zoff[s + 1] = lat.zoff[s] + zs;
    }
    lat.Z = lat.zoff[n_shells];
    if (lat.Z > kMaxZ) return "internal: shell sizes exceed kMaxZ";

    for (int b = 0; b < lat.A; ++b)
        for (int e = 0; e < lat.Z; ++e) {
            const Vec q = {bs[b].x + offs[e][0], bs[b].y + offs[e][1], bs[b].z + offs[e][2]};
            const int nb = basis_by_parity(type, lat.A, q);
            if (nb < 0) return "internal: offset leaves the lattice";
            // (q - basis[nb]) is even in every component, so the division is exact also for negatives.
            lat.stencil[b][e] = {(int8_t)nb, (int8_t)((q.x - bs[nb].x) / 2), (int8_t)((q.y - bs[nb].y) / 2),
                                 (int8_t)((q.z - bs[nb].z) / 2)};
        }
    return "";
}

static void fill_range(const Lattice& lat, int64_t first, int64_t last, int e0, int e1, int32_t* out)
{
    const int A = lat.A, Lx = lat.L[0], Ly = lat.L[1], Lz = lat.L[2];
    const int width = e1 - e0;
    for (int64_t site = first; site < last; ++site) {
        const int b = (int)(site % A);
        int64_t cell = site / A;
        const int cz = (int)(cell % Lz); cell /= Lz;
        const int cy = (int)(cell % Ly);
        const int cx = (int)(cell / Ly);
        int32_t* row = out + (site - first) * width;
        for (int e = e0; e < e1; ++e) {
            const StencilEntry& st = lat.stencil[b][e];
            const int nx = wrap(cx + st.sx, Lx), ny = wrap(cy + st.sy, Ly), nz = wrap(cz + st.sz, Lz);
            row[e - e0] = (int32_t)((((int64_t)nx * Ly + ny) * Lz + nz) * A + st.nb);
        }
    }
}

static void fill_parallel(const Lattice& lat, int64_t first, int64_t last, int e0, int e1, int32_t* out)
{
    const int64_t n = last - first;
    unsigned hw = std::thread::hardware_concurrency();
    int nt = (int)std::min<int64_t>(hw ? hw : 1, std::max<int64_t>(1, n / 65536));
    if (nt <= 1) { fill_range(lat, first, last, e0, e1, out); return; }
    std::vector<std::thread> th;
    const int width = e1 - e0;
    for (int t = 0; t < nt; ++t) {
        const int64_t a = first + n * t / nt, b = first + n * (t + 1) / nt;
        th.emplace_back([&lat, a, b, e0, e1, out, first, width] { fill_range(lat, a, b, e0, e1, out + (a - first) * width); });
    }
    for (auto& t : th) t.join();
}

void build_site_major(const Lattice& lat, int64_t first, int64_t last, int32_t* out)
{
    fill_parallel(lat, first, last, 0, lat.Z, out);
}

void build_shell_table(const Lattice& lat, int shell, int32_t* out)
{
    fill_parallel(lat, 0, lat.N, lat.zoff[shell], lat.zoff[shell + 1], out);
}

std::string species_counts(int64_t N, int M, const double* conc, int64_t* out)
{
    // D3, written as a ranking: every species first gets the integer part of c_i N (or c_i N itself when that is an
    // integer to 1e-9); the atoms still missing go, one each, to the species ranked by remainder, largest first,
    // equal remainders in index order (a stable sort keeps the index order).
    struct Share { int species; double remainder; };
    std::vector<Share> rank;
    double conc_sum = 0.0;
    int64_t placed = 0;
    for (int i = 0; i < M; ++i) {
        if (!(conc[i] > 0.0)) return "concentrations must be > 0";
        conc_sum += conc[i];
        const double want = conc[i] * (double)N;
        const double whole = std::nearbyint(want);
        if (std::fabs(want - whole) <= 1e-9) {
            out[i] = (int64_t)whole;
        } else {
            out[i] = (int64_t)std::floor(want);
            rank.push_back({i, want - std::floor(want)});
        }
        placed += out[i];
    }
    if (std::fabs(conc_sum - 1.0) > 1e-9) return "concentrations must sum to 1 (within 1e-9)";
    const int64_t missing = N - placed;
    if (missing < 0 || missing > (int64_t)rank.size()) return "species counts do not add up to N";
    std::stable_sort(rank.begin(), rank.end(), [](const Share& a, const Share& b) { return a.remainder > b.remainder; });
    for (int64_t r = 0; r < missing; ++r) ++out[rank[(size_t)r].species];
    for (int i = 0; i < M; ++i) if (out[i] <= 0) return "a species would get zero atoms";
    return "";
}

}  // namespace hea
