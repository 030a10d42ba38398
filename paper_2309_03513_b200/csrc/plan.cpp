#include "plan.h"
#include <algorithm>
#include <cmath>
#include <cstring>

namespace tddft {

void fft_plan_radices(int n, int* r1, int* r2, int* r3);
void scrambled_order_host(int N, int R1, int R2, int R3, int* freq_at_pos);

void reciprocal_lattice(const double* A, double* B, double* omega) {
    // rows b_i with b_i . a_j = 2 pi delta_ij  (b1 = 2 pi a2 x a3 / det, ...)
    const double* a1 = A; const double* a2 = A + 3; const double* a3 = A + 6;
    double c23[3] = {a2[1] * a3[2] - a2[2] * a3[1], a2[2] * a3[0] - a2[0] * a3[2], a2[0] * a3[1] - a2[1] * a3[0]};
    double c31[3] = {a3[1] * a1[2] - a3[2] * a1[1], a3[2] * a1[0] - a3[0] * a1[2], a3[0] * a1[1] - a3[1] * a1[0]};
    double c12[3] = {a1[1] * a2[2] - a1[2] * a2[1], a1[2] * a2[0] - a1[0] * a2[2], a1[0] * a2[1] - a1[1] * a2[0]};
    double det = a1[0] * c23[0] + a1[1] * c23[1] + a1[2] * c23[2];
    const double tp = 2.0 * M_PI;
    for (int i = 0; i < 3; ++i) { B[i] = tp * c23[i] / det; B[3 + i] = tp * c31[i] / det; B[6 + i] = tp * c12[i] / det; }
    *omega = std::fabs(det);
}

struct GEntry { double g2; int m[3]; int shell; };

long enumerate_half_sphere(const double* A, double ecut, std::vector<int>* miller, std::vector<double>* g2out) {
    double B[9], omega;
    reciprocal_lattice(A, B, &omega);
    const double gmax = std::sqrt(ecut);
    int bound[3];
    for (int i = 0; i < 3; ++i) {
        double len = std::sqrt(A[3 * i] * A[3 * i] + A[3 * i + 1] * A[3 * i + 1] + A[3 * i + 2] * A[3 * i + 2]);
        bound[i] = (int)std::floor(gmax * len / (2.0 * M_PI)) + 1;
    }
    std::vector<GEntry> list;
    for (int m1 = 0; m1 <= bound[0]; ++m1)
        for (int m2 = -bound[1]; m2 <= bound[1]; ++m2)
            for (int m3 = -bound[2]; m3 <= bound[2]; ++m3) {
                if (m1 == 0 && (m2 < 0 || (m2 == 0 && m3 < 0))) continue;
                double gx = m1 * B[0] + m2 * B[3] + m3 * B[6];
                double gy = m1 * B[1] + m2 * B[4] + m3 * B[7];
                double gz = m1 * B[2] + m2 * B[5] + m3 * B[8];
                double q = gx * gx + gy * gy + gz * gz;
                if (q <= ecut) list.push_back(GEntry{q, {m1, m2, m3}, 0});
            }
    std::stable_sort(list.begin(), list.end(), [](const GEntry& a, const GEntry& b) { return a.g2 < b.g2; });
    int shell = 0;
    for (size_t i = 0; i < list.size(); ++i) {
        if (i > 0 && list[i].g2 - list[i - 1].g2 > 1e-12 * list[i].g2) ++shell;
        list[i].shell = shell;
    }
    std::sort(list.begin(), list.end(), [](const GEntry& a, const GEntry& b) {
        if (a.shell != b.shell) return a.shell < b.shell;
        if (a.m[0] != b.m[0]) return a.m[0] < b.m[0];
        if (a.m[1] != b.m[1]) return a.m[1] < b.m[1];
        return a.m[2] < b.m[2];
    });
    if (miller) { miller->resize(3 * list.size()); for (size_t i = 0; i < list.size(); ++i) for (int c = 0; c < 3; ++c) (*miller)[3 * i + c] = list[i].m[c]; }
    if (g2out) { g2out->resize(list.size()); for (size_t i = 0; i < list.size(); ++i) (*g2out)[i] = list[i].g2; }
    return (long)list.size();
}

static void scramble(int n, const int* r, int nr, int* out) {
    // position p = k1*(n/R) + p', frequency k = R*k' + k1 (forward decimation in frequency, radix R first)
    if (nr == 0 || n == 1) { out[0] = 0; return; }
    const int R = r[0], M = n / R;
    std::vector<int> sub(M);
    scramble(M, r + 1, nr - 1, sub.data());
    for (int k1 = 0; k1 < R; ++k1) for (int p = 0; p < M; ++p) out[k1 * M + p] = R * sub[p] + k1;
}

const char* build_host_plan(const double* A, const int* grid, double ecut, HostPlan* hp) {
    std::memcpy(hp->A, A, 9 * sizeof(double));
    reciprocal_lattice(A, hp->B, &hp->omega);
    if (!(hp->omega > 0)) return "lattice is singular";
    for (int a = 0; a < 3; ++a) hp->n[a] = grid[a];
    hp->nr = (long)grid[0] * grid[1] * grid[2];
    hp->npwh = enumerate_half_sphere(A, ecut, &hp->miller, &hp->g2);
    int mmax[3] = {0, 0, 0};
    for (long g = 0; g < hp->npwh; ++g) for (int a = 0; a < 3; ++a) mmax[a] = std::max(mmax[a], std::abs(hp->miller[3 * g + a]));
    for (int a = 0; a < 3; ++a) if (2 * mmax[a] + 1 > grid[a]) return "FFT grid does not hold the plane-wave sphere (need 2*m_max+1 <= n)";
    for (int a = 0; a < 3; ++a) {
        int r[3];
        fft_plan_radices(grid[a], &r[0], &r[1], &r[2]);
        if (r[0] == 0) return "FFT length without a plan (supported: 2-3-5 smooth lengths listed in fft_core.cuh)";
        int nst = (r[1] == 1) ? 1 : (r[2] == 1 ? 2 : 3);
        std::vector<int> freq_at_pos(grid[a]);
        scramble(grid[a], r, nst, freq_at_pos.data());
        hp->pos[a].assign(grid[a], 0);
        for (int p = 0; p < grid[a]; ++p) hp->pos[a][freq_at_pos[p]] = p;
    }
    const int n1 = grid[0], n2 = grid[1], n3 = grid[2];
    auto flat = [&](int k1, int k2, int k3) { return ((long)hp->pos[0][k1] * n2 + hp->pos[1][k2]) * n3 + hp->pos[2][k3]; };
    auto wrap = [](int m, int n) { int j = m % n; return j < 0 ? j + n : j; };
    hp->idx_p.resize(hp->npwh); hp->idx_m.resize(hp->npwh);
    for (long g = 0; g < hp->npwh; ++g) {
        const int* m = &hp->miller[3 * g];
        hp->idx_p[g] = (int)flat(wrap(m[0], n1), wrap(m[1], n2), wrap(m[2], n3));
        hp->idx_m[g] = (int)flat(wrap(-m[0], n1), wrap(-m[1], n2), wrap(-m[2], n3));
    }
    // Coulomb table: signed Miller index m = j if j < (n+1)/2 else j - n (reading A7); value symmetrised over +-G so
    // that the potential of a real density is real on Nyquist planes of non-orthogonal cells (reading A17)
    auto sgn = [](int j, int n) { return j < (n + 1) / 2 ? j : j - n; };
    auto kval = [&](int j1, int j2, int j3) {
        const int m1 = sgn(j1, n1), m2 = sgn(j2, n2), m3 = sgn(j3, n3);
        double gx = m1 * hp->B[0] + m2 * hp->B[3] + m3 * hp->B[6];
        double gy = m1 * hp->B[1] + m2 * hp->B[4] + m3 * hp->B[7];
        double gz = m1 * hp->B[2] + m2 * hp->B[5] + m3 * hp->B[8];
        double q = gx * gx + gy * gy + gz * gz;
        return q > 0 ? 4.0 * M_PI / q : 0.0;
    };
    hp->vc.assign(hp->nr, 0.0);
    const double inv_nr = 1.0 / (double)hp->nr;
    for (int j1 = 0; j1 < n1; ++j1) for (int j2 = 0; j2 < n2; ++j2) for (int j3 = 0; j3 < n3; ++j3) {
        if (j1 == 0 && j2 == 0 && j3 == 0) continue;
        double k = 0.5 * (kval(j1, j2, j3) + kval((n1 - j1) % n1, (n2 - j2) % n2, (n3 - j3) % n3));
        hp->vc[flat(j1, j2, j3)] = k * inv_nr;
    }
    // pruned layouts of the fused path (plan.h)
    for (int kind = 0; kind < 2; ++kind) {
        const double rad2 = (kind == 0 ? 4.0 : 1.0) * ecut * (1.0 + 1e-9);
        const double gmax = std::sqrt(rad2);
        int mb[3];
        for (int i = 0; i < 3; ++i) {
            double len = std::sqrt(A[3 * i] * A[3 * i] + A[3 * i + 1] * A[3 * i + 1] + A[3 * i + 2] * A[3 * i + 2]);
            mb[i] = (int)std::floor(gmax * len / (2.0 * M_PI)) + 1;
        }
        std::vector<char> live((size_t)n2 * n3, 0);
        for (int m1 = -mb[0]; m1 <= mb[0]; ++m1) for (int m2 = -mb[1]; m2 <= mb[1]; ++m2) for (int m3 = -mb[2]; m3 <= mb[2]; ++m3) {
            double gx = m1 * hp->B[0] + m2 * hp->B[3] + m3 * hp->B[6];
            double gy = m1 * hp->B[1] + m2 * hp->B[4] + m3 * hp->B[7];
            double gz = m1 * hp->B[2] + m2 * hp->B[5] + m3 * hp->B[8];
            if (gx * gx + gy * gy + gz * gz <= rad2) live[(size_t)hp->pos[1][wrap(m2, n2)] * n3 + hp->pos[2][wrap(m3, n3)]] = 1;
        }
        hp->colmap[kind].assign((size_t)n2 * n3, -1);
        int nc = 0;
        for (size_t o = 0; o < live.size(); ++o) if (live[o]) hp->colmap[kind][o] = nc++;
        hp->ncols[kind] = nc;
    }
    {
        const int nc0 = hp->ncols[0], nc1 = hp->ncols[1];
        hp->vc_c.assign((size_t)n1 * nc0, 0.0);
        for (int xp = 0; xp < n1; ++xp) for (long o = 0; o < (long)n2 * n3; ++o) {
            const int cc = hp->colmap[0][o];
            if (cc >= 0) hp->vc_c[(size_t)xp * nc0 + cc] = hp->vc[(size_t)xp * n2 * n3 + o];
        }
        hp->idx_p_c.resize(hp->npwh); hp->idx_m_c.resize(hp->npwh);
        const long plane = (long)n2 * n3;
        for (long g = 0; g < hp->npwh; ++g) {
            const long ip = hp->idx_p[g], im = hp->idx_m[g];
            const int cp = hp->colmap[1][ip % plane], cm = hp->colmap[1][im % plane];
            if (cp < 0 || cm < 0) return "internal: sphere column outside the pruned layout";
            hp->idx_p_c[g] = (int)((ip / plane) * nc1 + cp);
            hp->idx_m_c[g] = (int)((im / plane) * nc1 + cm);
        }
    }
    return nullptr;
}

}  // namespace tddft
