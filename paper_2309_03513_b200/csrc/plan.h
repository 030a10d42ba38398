// Host-side plan: reciprocal lattice, canonical plane-wave half sphere, scrambled FFT index maps and the
// Coulomb table.  Pure host code.
#pragma once
#include <vector>

namespace tddft {

struct HostPlan {
    double A[9], B[9], omega;
    int n[3];
    long nr;
    long npwh;
    std::vector<int> miller;       // [npwh][3]
    std::vector<double> g2;        // [npwh] |G|^2 (bohr^-2)
    std::vector<int> pos[3];       // pos[a][k] = position of frequency index k (0..n-1) along axis a after the forward DIF
    std::vector<int> idx_p, idx_m; // [npwh] scrambled flat positions of G and -G
    std::vector<double> vc;        // [nr] symmetrised 4 pi/|G|^2 / N_r in scrambled layout, G = 0 -> 0
    // Pruned frequency-space layout of the fused FFT path.  A function whose plane waves lie inside the sphere has
    // non-zero (ky,kz) columns only where the sphere's shadow falls; a product of two such functions (a pair density
    // phi_v phi_v', or a response density, Eq. 4) only inside the shadow of the sphere of twice the
    // radius (wrapped onto the grid where it aliases, reading A13).  Work grids keep live columns only:
    // element (x position, column c) at x*ncols + c, c numbering the live (ypos*n3 + zpos) in ascending order.
    // kind 0 = products (radius 2 sqrt(ecut)), kind 1 = sphere functions (radius sqrt(ecut)).
    int ncols[2];
    std::vector<int> colmap[2];    // [n2*n3] scrambled plane offset -> compact column, -1 = dead
    std::vector<int> idx_p_c, idx_m_c;   // [npwh] compact (kind 1) positions of G and -G
    std::vector<double> vc_c;      // [n1][ncols[0]] the Coulomb table on the kind-0 columns
};

void reciprocal_lattice(const double* A, double* B, double* omega);
// reading A7; returns the count, fills miller/g2 if non-null
long enumerate_half_sphere(const double* A, double ecut_ry, std::vector<int>* miller, std::vector<double>* g2);
// returns empty string or an error message
const char* build_host_plan(const double* A, const int* grid, double ecut_ry, HostPlan* hp);

}  // namespace tddft
