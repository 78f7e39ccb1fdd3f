// Host-side tables of the DOCTORS hot path: quadrature, real spherical harmonics,
// projection tables and the integer sweep schedules.  Plain C++ (no CUDA).
#pragma once
#include <cstdint>
#include <vector>

namespace doctors {

// Level-symmetric LQ_N (PAPER.md:39-42, :208 give only N(N+2); the rule is DESIGN.md App. A).
// omega [n][3], w [n], sum w = 4 pi; octant-major, octant bit0/1/2 = negative x/y/z.
bool level_symmetric(int N, std::vector<double>& omega, std::vector<double>& w);

// Real harmonics of reading R4 in Cartesian form, l <= 3.  Y has (L+1)^2 entries.
void real_harmonics(int L, double mu, double eta, double xi, double* Y);

// Mtab [n][nm] = (2l+1)/(4 pi) Y_lm(Omega_n)  (moment -> direction, Eq. 2 rhs in moment form)
// Dtab [n][nm] = w_n Y_lm(Omega_n)            (direction -> moment, Eq. 3)
void projection_tables(int L, const std::vector<double>& omega, const std::vector<double>& w,
                       std::vector<double>& Mtab, std::vector<double>& Dtab);

// P(S), Eqs. (9)-(22).
long long wavefront_size(int nx, int ny, int nz, int S);

// Sub-sweep schedule, PAPER.md:72-81 (Eq. 8) in Table 1 order, mirrored per
// octant.  plane_offset: nx+ny+nz-1 entries; cell_of: nx*ny*nz entries, index i + nx*(j + ny*k).
void subsweep_schedule(int nx, int ny, int nz, int octant,
                       std::vector<int32_t>& plane_offset, std::vector<int32_t>& cell_of);

}  // namespace doctors
