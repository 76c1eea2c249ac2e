// hea_lattice.hpp -- host-side lattice description and shell neighbour-table builder (product code; shares nothing
// with oracle/).  DESIGN.md D1-D3; PAPER.md P:105 (supercell S = A*L^3, 3 coordination shells), P:256-262 (shells k).
//
// The builder works from a STENCIL: for a site with basis index b, entry k of the concatenated shell list leads to
// basis index nb[b][k] in the cell shifted by (sx, sy, sz)[b][k] conventional cells.  The same stencil drives the
// host table builder and the table-free neighbour computation inside the MC kernel.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace hea {

constexpr int kMaxSpecies = 8;
constexpr int kMaxShells = 3;
constexpr int kMaxBasis = 4;
constexpr int kMaxZ = 42;                 // 12 + 6 + 24 (fcc, 3 shells); bcc: 8 + 6 + 12 = 26

struct StencilEntry { int8_t nb, sx, sy, sz; };

struct Lattice {
    int type = 0;                         // 0 fcc, 1 bcc
    int L[3] = {0, 0, 0};
    int A = 0;                            // basis size
    int64_t N = 0;
    int S = 0;
    int z[kMaxShells] = {0, 0, 0};
    int zoff[kMaxShells + 1] = {0, 0, 0, 0};
    int Z = 0;                            // sum of z
    StencilEntry stencil[kMaxBasis][kMaxZ];
};

// Fills `lat` (shell sizes, stencil).  Returns empty string on success, else an error message.
std::string lattice_init(Lattice& lat, int type, int Lx, int Ly, int Lz, int n_shells);

// Neighbour entries [first, last) of the site-major table: out[(site - first) * Z + e], e over concatenated shells.
void build_site_major(const Lattice& lat, int64_t first, int64_t last, int32_t* out);

// One shell, [N][z_shell], for hea_neighbor_table.
void build_shell_table(const Lattice& lat, int shell, int32_t* out);

// D3: species counts from concentrations.  Returns empty string on success.
std::string species_counts(int64_t N, int M, const double* conc, int64_t* out);

}  // namespace hea
