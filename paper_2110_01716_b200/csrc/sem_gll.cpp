// sem_gll.cpp — host-side 1-D GLL data for order N (a0; "GLL quadrature points", P:93 D_il = dh_l/dr at xi_i).
// Product code, independent of oracle/: nodes by Newton on P_N' using the derivative recurrences, weights from
// 2/(N(N+1)P_N^2), and D from the barycentric form of the Lagrange derivative with the negative-sum diagonal.
#include <cmath>

#include "sem_internal.h"

namespace {
// P_n(x), P_n'(x), P_n''(x) by the Bonnet recurrence and its two derivatives.
void legendre3(int n, long double x, long double& P, long double& dP, long double& d2P) {
    long double a0 = 1, a1 = x, b0 = 0, b1 = 1, c0 = 0, c1 = 0;
    if (n == 0) { P = 1; dP = 0; d2P = 0; return; }
    for (int m = 1; m < n; ++m) {
        const long double f = (2.0L * m + 1.0L) / (m + 1.0L), g = (long double)m / (m + 1.0L);
        const long double a2 = f * x * a1 - g * a0;
        const long double b2 = f * (a1 + x * b1) - g * b0;
        const long double c2 = f * (2.0L * b1 + x * c1) - g * c0;
        a0 = a1; a1 = a2; b0 = b1; b1 = b2; c0 = c1; c1 = c2;
    }
    P = a1; dP = b1; d2P = c1;
}
}  // namespace

void sem_gll_tables(int N, double* xi, double* rho, double* D) {
    const int p = N + 1;
    long double x[SEM_MAXP], bw[SEM_MAXP];
    const long double pi = acosl(-1.0L);
    for (int i = 0; i < p; ++i) {
        if (i == 0) { x[i] = -1.0L; continue; }
        if (i == N) { x[i] = 1.0L; continue; }
        if (2 * i == N) { x[i] = 0.0L; continue; }
        if (2 * i > N) { x[i] = -x[N - i]; continue; }     // the node set is symmetric about 0
        long double t = -cosl(pi * i / N);
        for (int it = 0; it < 60; ++it) {
            long double P, dP, d2P;
            legendre3(N, t, P, dP, d2P);
            const long double step = dP / d2P;
            t -= step;
            if (fabsl(step) < 1e-20L) break;
        }
        x[i] = t;
    }
    for (int i = 0; i < p; ++i) {
        long double P, dP, d2P;
        legendre3(N, x[i], P, dP, d2P);
        xi[i] = (double)x[i];
        rho[i] = (double)(2.0L / ((long double)N * (N + 1) * P * P));
        long double prod = 1.0L;
        for (int j = 0; j < p; ++j)
            if (j != i) prod *= (x[i] - x[j]);
        bw[i] = 1.0L / prod;                                // barycentric weight of node i
    }
    for (int i = 0; i < p; ++i) {
        long double diag = 0.0L;
        for (int l = 0; l < p; ++l) {
            if (l == i) continue;
            const long double d = (bw[l] / bw[i]) / (x[i] - x[l]);
            D[i * p + l] = (double)d;
            diag -= d;                                       // rows of D annihilate constants
        }
        D[i * p + i] = (double)diag;
    }
    // interior diagonal entries are exactly zero in exact arithmetic; the negative sum leaves O(1e-19) noise that
    // rounds to a tiny double — keep it (it is the correctly rounded row-sum-zero value).
}
