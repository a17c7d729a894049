// adft_sph.cuh -- Cartesian -> real-solid-harmonic transformation of an N x N matrix (J, K): SURVEY.md 8(f4)
// "spherical-harmonic output".  M_sph = T^T M_cart T, T block diagonal over the shells.
//
// The real solid harmonics are TABULATED here as integer polynomials in x, y, z (the textbook forms up to g), in the
// order m = -l, ..., +l; each is scaled on the host to unit norm under the overlap of the shell's Cartesian components,
//   <x^a y^b z^c | x^a' y^b' z^c'> = (a+a'-1)!! (b+b'-1)!! (c+c'-1)!! / (2L-1)!!   (all sums even, else 0),
// which holds for every exponent and contraction because all components of a shell share one radial function
// (R-1: unit self-overlap of the (L,0,0) component).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace adft {

constexpr int SPH_LMAX = 4, SPH_NCART_MAX = 15, SPH_NSPH_MAX = 9;

struct SphTerm { int8_t a, b, c; int16_t coef; };
struct SphPoly { int nterm; SphTerm t[9]; };

// S_lm, m = -l..l (unnormalised; r^2 = xx + yy + zz expanded)
static const SphPoly SPH_TABLE[SPH_LMAX + 1][SPH_NSPH_MAX] = {
    /* l = 0 */ {{1, {{0, 0, 0, 1}}}},
    /* l = 1 */ {{1, {{0, 1, 0, 1}}}, {1, {{0, 0, 1, 1}}}, {1, {{1, 0, 0, 1}}}},
    /* l = 2 */ {{1, {{1, 1, 0, 1}}},                                               // xy
                 {1, {{0, 1, 1, 1}}},                                               // yz
                 {3, {{0, 0, 2, 2}, {2, 0, 0, -1}, {0, 2, 0, -1}}},                 // 2zz - xx - yy
                 {1, {{1, 0, 1, 1}}},                                               // xz
                 {2, {{2, 0, 0, 1}, {0, 2, 0, -1}}}},                               // xx - yy
    /* l = 3 */ {{2, {{2, 1, 0, 3}, {0, 3, 0, -1}}},                                // 3xxy - yyy
                 {1, {{1, 1, 1, 1}}},                                               // xyz
                 {3, {{0, 1, 2, 4}, {2, 1, 0, -1}, {0, 3, 0, -1}}},                 // y(4zz - xx - yy)
                 {3, {{0, 0, 3, 2}, {2, 0, 1, -3}, {0, 2, 1, -3}}},                 // z(2zz - 3xx - 3yy)
                 {3, {{1, 0, 2, 4}, {3, 0, 0, -1}, {1, 2, 0, -1}}},                 // x(4zz - xx - yy)
                 {2, {{2, 0, 1, 1}, {0, 2, 1, -1}}},                                // z(xx - yy)
                 {2, {{3, 0, 0, 1}, {1, 2, 0, -3}}}},                               // xxx - 3xyy
    /* l = 4 */ {{2, {{3, 1, 0, 1}, {1, 3, 0, -1}}},                                // xy(xx - yy)
                 {2, {{2, 1, 1, 3}, {0, 3, 1, -1}}},                                // yz(3xx - yy)
                 {3, {{1, 1, 2, 6}, {3, 1, 0, -1}, {1, 3, 0, -1}}},                 // xy(6zz - xx - yy)
                 {3, {{0, 1, 3, 4}, {2, 1, 1, -3}, {0, 3, 1, -3}}},                 // yz(4zz - 3xx - 3yy)
                 {6, {{0, 0, 4, 8}, {2, 0, 2, -24}, {0, 2, 2, -24}, {4, 0, 0, 3}, {2, 2, 0, 6}, {0, 4, 0, 3}}},   // 35z^4 - 30z^2r^2 + 3r^4
                 {3, {{1, 0, 3, 4}, {3, 0, 1, -3}, {1, 2, 1, -3}}},                 // xz(4zz - 3xx - 3yy)
                 {4, {{2, 0, 2, 6}, {0, 2, 2, -6}, {4, 0, 0, -1}, {0, 4, 0, 1}}},   // (xx - yy)(6zz - xx - yy)
                 {2, {{3, 0, 1, 1}, {1, 2, 1, -3}}},                                // xz(xx - 3yy)
                 {3, {{4, 0, 0, 1}, {2, 2, 0, -6}, {0, 4, 0, 1}}}},                 // x^4 - 6xxyy + y^4
};

// T[l][cart][m + l], filled by sph_fill_tables() and copied to the device once per pairs handle
struct SphTables { double T[SPH_LMAX + 1][SPH_NCART_MAX][SPH_NSPH_MAX]; };

inline int sph_cart_index(int l, int a, int b)          // position of (a, b, l-a-b) in the component order of DESIGN.md R-3
{
    int idx = 0;
    for (int x = l; x >= 0; --x)
        for (int y = l - x; y >= 0; --y) {
            if (x == a && y == b) return idx;
            ++idx;
        }
    return -1;
}
inline double sph_dfact(int n) { double r = 1.0; for (; n > 1; n -= 2) r *= n; return r; }

inline void sph_fill_tables(SphTables &tab)
{
    for (int l = 0; l <= SPH_LMAX; ++l) {
        const int nc = (l + 1) * (l + 2) / 2;
        int ca[SPH_NCART_MAX][3];
        for (int x = l, n = 0; x >= 0; --x)
            for (int y = l - x; y >= 0; --y, ++n) { ca[n][0] = x; ca[n][1] = y; ca[n][2] = l - x - y; }
        for (int m = 0; m < 2 * l + 1; ++m) {
            double v[SPH_NCART_MAX] = {};
            const SphPoly &p = SPH_TABLE[l][m];
            for (int k = 0; k < p.nterm; ++k) v[sph_cart_index(l, p.t[k].a, p.t[k].b)] += p.t[k].coef;
            double nrm = 0.0;
            for (int i = 0; i < nc; ++i)
                for (int j = 0; j < nc; ++j) {
                    const int s0 = ca[i][0] + ca[j][0], s1 = ca[i][1] + ca[j][1], s2 = ca[i][2] + ca[j][2];
                    if ((s0 | s1 | s2) & 1) continue;
                    nrm += v[i] * v[j] * sph_dfact(s0 - 1) * sph_dfact(s1 - 1) * sph_dfact(s2 - 1) / sph_dfact(2 * l - 1);
                }
            for (int i = 0; i < SPH_NCART_MAX; ++i) tab.T[l][i][m] = i < nc ? v[i] / sqrt(nrm) : 0.0;
        }
    }
}

// out[i, j] = sum_{a in shell(i), b in shell(j)} T[a, m_i] M[a, b] T[b, m_j]; one thread per element of M_sph.
// sph_shell[i], sph_m[i]: shell and m + l of spherical function i; bfoff: first Cartesian function of a shell.
__global__ void cart_to_sph_kernel(const double *__restrict__ M, int N, double *__restrict__ out, int Ns,
                                   const int32_t *__restrict__ sph_shell, const int32_t *__restrict__ sph_m,
                                   const int32_t *__restrict__ bfoff, const int32_t *__restrict__ shell_l,
                                   const SphTables *__restrict__ tab)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= Ns || j >= Ns) return;
    const int A = sph_shell[i], B = sph_shell[j], ma = sph_m[i], mb = sph_m[j];
    const int la = shell_l[A], lb = shell_l[B];
    const int a0 = bfoff[A], b0 = bfoff[B], na = (la + 1) * (la + 2) / 2, nb = (lb + 1) * (lb + 2) / 2;
    double s = 0.0;
    for (int a = 0; a < na; ++a) {
        const double ta = tab->T[la][a][ma];
        if (ta == 0.0) continue;
        double r = 0.0;
        for (int b = 0; b < nb; ++b) r = fma(tab->T[lb][b][mb], __ldg(M + (size_t)(a0 + a) * N + b0 + b), r);
        s = fma(ta, r, s);
    }
    out[(size_t)i * Ns + j] = s;
}

}  // namespace adft
