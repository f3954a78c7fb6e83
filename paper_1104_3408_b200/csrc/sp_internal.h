// Internal header of libspshell (not part of the ABI; the oracle never includes it).
#pragma once
#include <vector>

struct SpHostMatrices {
    int Nr = 0, Nt = 0, Np = 0, L = 0;
    double rin = 0, rout = 0;
    std::vector<double> cd;    // CD^ [Nr][Nr] row-major                       (eq. 9)
    std::vector<double> g2;    // FD_{2Nt}[i][i'] = g2[(i-i') mod 2Nt]         (eq. 8; circulant)
    std::vector<double> g3;    // FD_{Np}[j][j']  = g3[(j-j') mod Np]
    std::vector<double> an;    // Fourier analysis  [2L+1][Np]                 (eq. 24; rows a_0, a_1, b_1, a_2, ...)
    std::vector<double> sy;    // Fourier synthesis [Np][2L+1]                 (eq. 23; same column order)
    std::vector<double> F;     // F^n_m [7][L+1][Nt][Nt], n = -3..3            (eq. 62)
    std::vector<double> r, inv_r, sin_t, cos_t, inv_sin_t, sin_p, cos_p;      // grid / Jacobian factors (eq. 2-4, 6)
};

// Host construction in extended precision (long double / binary128), rounded once to double.
void sp_host_build(int Nr, int Nt, int Np, double rin, double rout, int L, SpHostMatrices &out);
