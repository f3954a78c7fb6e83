// Host-side matrix construction for libspshell (start-up cost only: PAPER.md:43, 114, 215, 289).
//
// Route (deliberately the PAPER'S, and different from the test oracle's): spin-weighted associated
// Legendre functions by the n-recursion (42)-(44) starting from ordinary normalised associated
// Legendre functions, evaluated in binary128 because the recursion loses up to 5e-10 in double near
// the poles (1/sin^3 cancellation); pseudo-inverse by a one-sided Jacobi SVD in long
// double; F^n_m = P f_diag P^+ (eq. 62); everything rounded once to double.
#include "sp_internal.h"

#include <quadmath.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <thread>

typedef __float128 q128;
typedef long double ld;

static const q128 PI_Q = M_PIq;

// Ordinary orthonormal associated Legendre functions Phat_l^m(cos th), 0 <= m <= l <= lmax (eq. 26),
// stable three-term recurrence in l.  out[m*(lmax+1)+l].
static void legendre_hat(int lmax, q128 th, std::vector<q128> &out) {
    q128 x = cosq(th), s = sinq(th);
    int w = lmax + 1;
    out.assign((size_t)w * w, 0);
    q128 pmm = sqrtq(1 / (4 * PI_Q));
    for (int m = 0; m <= lmax; m++) {
        if (m > 0) pmm = -sqrtq((q128)(2 * m + 1) / (q128)(2 * m)) * s * pmm;
        out[(size_t)m * w + m] = pmm;
        if (m + 1 <= lmax) out[(size_t)m * w + m + 1] = sqrtq((q128)(2 * m + 3)) * x * pmm;
        for (int l = m + 2; l <= lmax; l++) {
            q128 a = sqrtq((q128)(4 * l * l - 1) / (q128)(l * l - m * m));
            q128 b = sqrtq((q128)((l - 1) * (l - 1) - m * m) / (q128)(4 * (l - 1) * (l - 1) - 1));
            out[(size_t)m * w + l] = a * (x * out[(size_t)m * w + l - 1] - b * out[(size_t)m * w + l - 2]);
        }
    }
}

// P^n_{lm}(th) for n = 0..3, m = -lmax..lmax, l = 0..lmax by eq. (42)-(44).  Y[n][(m+lmax)*(lmax+1)+l].
static void spin_legendre_up(int lmax, q128 th, std::vector<q128> Y[4]) {
    int w = lmax + 1, nm = 2 * lmax + 1;
    std::vector<q128> P0;
    legendre_hat(lmax, th, P0);
    q128 c = cosq(th), s = sinq(th);
    Y[0].assign((size_t)nm * w, 0);
    for (int m = -lmax; m <= lmax; m++) {
        int am = m < 0 ? -m : m;
        q128 sg = (m < 0 && (am & 1)) ? -1 : 1;                    // eq. 47 with n = 0
        for (int l = am; l <= lmax; l++) Y[0][(size_t)(m + lmax) * w + l] = sg * P0[(size_t)am * w + l];
    }
    for (int n = 1; n <= 3; n++) {
        Y[n].assign((size_t)nm * w, 0);
        for (int m = -lmax; m <= lmax; m++) {
            const q128 *prev = &Y[n - 1][(size_t)(m + lmax) * w];
            q128 *cur = &Y[n][(size_t)(m + lmax) * w];
            int am = m < 0 ? -m : m;
            for (int l = std::max(n, am); l <= lmax; l++) {
                q128 alpha = sqrtq((q128)(l - n + 1) / (q128)(l + n));
                q128 beta = sqrtq((q128)(2 * l + 1) / (q128)(2 * l - 1) * (q128)(l + n - 1) * (q128)(l * l - m * m) / (q128)(l + n)) / l;
                cur[l] = alpha * ((q128)m / l - c) / s * prev[l] + beta / s * (l >= 1 ? prev[l - 1] : 0);
            }
        }
    }
}

// One-sided Jacobi (Hestenes) SVD of A (rows x cols, rows >= cols, row-major): on return W = U*Sigma
// (columns orthogonal), V orthogonal with A V = W.
static void jacobi_svd(int rows, int cols, std::vector<ld> &W, std::vector<ld> &V) {
    V.assign((size_t)cols * cols, 0);
    for (int c = 0; c < cols; c++) V[(size_t)c * cols + c] = 1;
    for (int sweep = 0; sweep < 60; sweep++) {
        ld off = 0;
        for (int p = 0; p < cols - 1; p++)
            for (int q = p + 1; q < cols; q++) {
                ld a = 0, b = 0, g = 0;
                for (int i = 0; i < rows; i++) {
                    ld x = W[(size_t)i * cols + p], y = W[(size_t)i * cols + q];
                    a += x * x; b += y * y; g += x * y;
                }
                if (a == 0 || b == 0) continue;
                ld rel = fabsl(g) / sqrtl(a * b);
                if (rel > off) off = rel;
                if (rel < 1e-19L) continue;
                ld zeta = (b - a) / (2 * g);
                ld t = (zeta >= 0 ? 1 : -1) / (fabsl(zeta) + sqrtl(1 + zeta * zeta));
                ld cs = 1 / sqrtl(1 + t * t), sn = cs * t;
                for (int i = 0; i < rows; i++) {
                    ld x = W[(size_t)i * cols + p], y = W[(size_t)i * cols + q];
                    W[(size_t)i * cols + p] = cs * x - sn * y;
                    W[(size_t)i * cols + q] = sn * x + cs * y;
                }
                for (int i = 0; i < cols; i++) {
                    ld x = V[(size_t)i * cols + p], y = V[(size_t)i * cols + q];
                    V[(size_t)i * cols + p] = cs * x - sn * y;
                    V[(size_t)i * cols + q] = sn * x + cs * y;
                }
            }
        if (off < 1e-18L) break;
    }
}

// F = P f P^+ (eq. 62), P: N x nc (columns l = l0..N-1), keep l <= L.  P^+ = V Sigma^-2 W^T.
static void filter_from_P(int N, int nc, int l0, int L, const std::vector<ld> &P, double *F) {
    std::vector<ld> W(P), V;
    jacobi_svd(N, nc, W, V);
    std::vector<ld> s2(nc);
    for (int c = 0; c < nc; c++) {
        ld a = 0;
        for (int i = 0; i < N; i++) a += W[(size_t)i * nc + c] * W[(size_t)i * nc + c];
        s2[c] = a;
    }
    // Pp[q][i] = sum_c V[q][c] W[i][c] / s2[c]
    std::vector<ld> Pp((size_t)nc * N);
    for (int q = 0; q < nc; q++)
        for (int i = 0; i < N; i++) {
            ld a = 0;
            for (int c = 0; c < nc; c++) a += V[(size_t)q * nc + c] * W[(size_t)i * nc + c] / s2[c];
            Pp[(size_t)q * N + i] = a;
        }
    for (int i = 0; i < N; i++)
        for (int ii = 0; ii < N; ii++) {
            ld a = 0;
            for (int q = 0; q < nc && l0 + q <= L; q++) a += P[(size_t)i * nc + q] * Pp[(size_t)q * N + ii];
            F[(size_t)i * N + ii] = (double)a;
        }
}

void sp_host_build(int Nr, int Nt, int Np, double rin, double rout, int L, SpHostMatrices &M) {
    M.Nr = Nr; M.Nt = Nt; M.Np = Np; M.L = L; M.rin = rin; M.rout = rout;
    const int N = Nt;
    // ---- grid and Jacobian factors (eq. 2-4, 6)
    M.r.resize(Nr); M.inv_r.resize(Nr);
    for (int k = 0; k < Nr; k++) {
        q128 r = ((q128)rout + (q128)rin) / 2 - ((q128)rout - (q128)rin) / 2 * cosq(PI_Q * k / (Nr - 1));
        M.r[k] = (double)r; M.inv_r[k] = (double)(1 / r);
    }
    M.sin_t.resize(Nt); M.cos_t.resize(Nt); M.inv_sin_t.resize(Nt);
    for (int i = 0; i < Nt; i++) {
        q128 th = PI_Q * (2 * i + 1) / (2 * Nt);
        M.sin_t[i] = (double)sinq(th); M.cos_t[i] = (double)cosq(th); M.inv_sin_t[i] = (double)(1 / sinq(th));
    }
    M.sin_p.resize(Np); M.cos_p.resize(Np);
    for (int j = 0; j < Np; j++) {
        q128 ph = 2 * PI_Q * j / Np;
        M.sin_p[j] = (double)sinq(ph); M.cos_p[j] = (double)cosq(ph);
    }
    // ---- CD^ (eq. 9): x_i - x_j = 2 sin((a_i+a_j)/2) sin((a_i-a_j)/2), a = pi i/(N-1); diagonal by negative row sum
    M.cd.assign((size_t)Nr * Nr, 0);
    {
        std::vector<q128> row(Nr);
        q128 scale = 2 / ((q128)rout - (q128)rin);
        for (int i = 0; i < Nr; i++) {
            q128 diag = 0;
            for (int j = 0; j < Nr; j++) {
                if (j == i) continue;
                q128 ci = (i == 0 || i == Nr - 1) ? 2 : 1, cj = (j == 0 || j == Nr - 1) ? 2 : 1;
                q128 dx = 2 * sinq(PI_Q * (i + j) / (2 * (Nr - 1))) * sinq(PI_Q * (i - j) / (2 * (Nr - 1)));
                row[j] = (ci / cj) * (((i + j) & 1) ? -1 : 1) / dx;
                diag -= row[j];
            }
            row[i] = diag;
            for (int j = 0; j < Nr; j++) M.cd[(size_t)i * Nr + j] = (double)(scale * row[j]);
        }
    }
    // ---- FD (eq. 8), circulant: g(d) = (-1)^d cot(d pi/n)/2, g(0) = 0
    auto fd = [](int n, std::vector<double> &g) {
        g.assign(n, 0);
        for (int d = 1; d < n; d++) {
            q128 a = PI_Q * d / n;
            g[d] = (double)(((d & 1) ? -1 : 1) * cosq(a) / (2 * sinq(a)));
        }
    };
    fd(2 * Nt, M.g2);
    fd(Np, M.g3);
    // ---- real Fourier analysis / synthesis (eq. 23-24, B = sin: reading Q1), modes m = 0..L
    const int MC = 2 * L + 1, J = Np;
    M.an.assign((size_t)MC * J, 0); M.sy.assign((size_t)J * MC, 0);
    for (int j = 0; j < J; j++) {
        M.an[j] = 1.0 / J; M.sy[(size_t)j * MC] = 1.0;
        for (int m = 1; m <= L; m++) {
            int qq = (int)(((long)m * j) % J);
            q128 a = 2 * PI_Q * qq / J;
            double c = (double)cosq(a), s = (double)sinq(a);
            double c2 = (double)(2 * cosq(a) / J), s2 = (double)(2 * sinq(a) / J);
            M.an[(size_t)(2 * m - 1) * J + j] = c2; M.an[(size_t)(2 * m) * J + j] = s2;
            M.sy[(size_t)j * MC + 2 * m - 1] = c; M.sy[(size_t)j * MC + 2 * m] = s;
        }
    }
    // ---- spin-weighted Legendre functions on the grid: Pq[n+3][m][i][l], m = 0..N-1
    const int lmax = N - 1, w = lmax + 1;
    std::vector<ld> Pn((size_t)7 * N * N * w, 0);
    auto PN = [&](int n, int m, int i, int l) -> ld & { return Pn[(((size_t)(n + 3) * N + m) * N + i) * w + l]; };
    {
        std::atomic<int> next(0);
        auto work = [&]() {
            std::vector<q128> Y[4];
            for (int i; (i = next.fetch_add(1)) < N;) {
                spin_legendre_up(lmax, PI_Q * (2 * i + 1) / (2 * N), Y);
                for (int n = 0; n <= 3; n++)
                    for (int m = 0; m <= lmax; m++)
                        for (int l = 0; l <= lmax; l++) {
                            PN(n, m, i, l) = (ld)Y[n][(size_t)(m + lmax) * w + l];
                            // eq. 47: P^{-n}_{l,m} = (-1)^{n+m} P^{n}_{l,-m}
                            if (n > 0) PN(-n, m, i, l) = (((n + m) & 1) ? -1 : 1) * (ld)Y[n][(size_t)(-m + lmax) * w + l];
                        }
            }
        };
        int nth = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
        std::vector<std::thread> th;
        for (int t = 0; t < nth; t++) th.emplace_back(work);
        for (auto &t : th) t.join();
    }
    // ---- F^n_m, n = -3..3, m = 0..L (eq. 48, 49, 62)
    M.F.assign((size_t)7 * (L + 1) * N * N, 0);
    {
        std::atomic<int> next(0);
        int total = 7 * (L + 1);
        auto work = [&]() {
            for (int it; (it = next.fetch_add(1)) < total;) {
                int n = it / (L + 1) - 3, m = it % (L + 1);
                int l0 = std::max(std::abs(n), m);
                if (l0 > L || l0 > N - 1) continue;
                int nc = N - l0;
                std::vector<ld> P((size_t)N * nc);
                for (int i = 0; i < N; i++)
                    for (int q = 0; q < nc; q++) P[(size_t)i * nc + q] = PN(n, m, i, l0 + q);
                filter_from_P(N, nc, l0, L, P, &M.F[(size_t)it * N * N]);
            }
        };
        int nth = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
        std::vector<std::thread> th;
        for (int t = 0; t < nth; t++) th.emplace_back(work);
        for (auto &t : th) t.join();
    }
}
