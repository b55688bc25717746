// sem_fdm_setup.cpp — NEXT-2a setup (host): the eigen-decompositions behind Eq. (3) ("fast diagonalization (FDM)
// Deville et al. (2002)").  For every element and direction d the 1-D pair (A_d stiffness, B_d mass; symmetric, B_d positive
// definite) is reduced to the generalised eigenproblem A_d s = lambda B_d s with S_d^T B_d S_d = I, S_d^T A_d S_d =
// diag(lambda_d); then Lambda[c][b][a] = lambda_x[a] + lambda_y[b] + lambda_z[c] (reading S28 in DESIGN.md).
// Method: Cholesky B = L L^T, C = L^-1 A L^-T, cyclic Jacobi rotations on C (m <= 16: a handful of sweeps to 1e-15),
// S = L^-T V, eigenvalues ascending.  Untimed setup, plain C++; elements are independent.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

#include "../../include/sem.h"

namespace {

constexpr int MAXM = 16;

// A, B: [m][m] row-major.  S: [m][m] eigenvectors in columns; lam[m] ascending.  false if B is not positive definite.
bool gen_eig(int m, const double* A, const double* B, double* S, double* lam) {
    double L[MAXM][MAXM] = {}, C[MAXM][MAXM], V[MAXM][MAXM], T[MAXM][MAXM];
    for (int i = 0; i < m; ++i)                               // Cholesky, lower
        for (int j = 0; j <= i; ++j) {
            double s = 0.5 * (B[i * m + j] + B[j * m + i]);
            for (int k = 0; k < j; ++k) s -= L[i][k] * L[j][k];
            if (i == j) {
                if (!(s > 0.0)) return false;
                L[i][i] = std::sqrt(s);
            } else {
                L[i][j] = s / L[j][j];
            }
        }
    for (int j = 0; j < m; ++j)                               // T = L^-1 A  (forward substitution per column)
        for (int i = 0; i < m; ++i) {
            double s = 0.5 * (A[i * m + j] + A[j * m + i]);
            for (int k = 0; k < i; ++k) s -= L[i][k] * T[k][j];
            T[i][j] = s / L[i][i];
        }
    for (int i = 0; i < m; ++i)                               // C = T L^-T: row i solves C[i][:] L^T = T[i][:]
        for (int j = 0; j < m; ++j) {
            double s = T[i][j];
            for (int k = 0; k < j; ++k) s -= C[i][k] * L[j][k];
            C[i][j] = s / L[j][j];
        }
    for (int i = 0; i < m; ++i)
        for (int j = 0; j < m; ++j) {
            if (j > i) C[i][j] = C[j][i] = 0.5 * (C[i][j] + C[j][i]);
            V[i][j] = i == j ? 1.0 : 0.0;
        }
    for (int sweep = 0; sweep < 60; ++sweep) {                // cyclic Jacobi
        double off = 0.0, dia = 0.0;
        for (int i = 0; i < m; ++i)
            for (int j = 0; j < m; ++j) (i == j ? dia : off) += C[i][j] * C[i][j];
        if (off <= 1e-32 * dia) break;
        for (int p = 0; p < m - 1; ++p)
            for (int q = p + 1; q < m; ++q) {
                if (C[p][q] == 0.0) continue;
                const double theta = (C[q][q] - C[p][p]) / (2.0 * C[p][q]);
                const double t = (theta >= 0.0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
                const double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
                for (int k = 0; k < m; ++k) {                 // columns p, q
                    const double a = C[k][p], b = C[k][q];
                    C[k][p] = c * a - s * b;
                    C[k][q] = s * a + c * b;
                }
                for (int k = 0; k < m; ++k) {                 // rows p, q
                    const double a = C[p][k], b = C[q][k];
                    C[p][k] = c * a - s * b;
                    C[q][k] = s * a + c * b;
                }
                for (int k = 0; k < m; ++k) {
                    const double a = V[k][p], b = V[k][q];
                    V[k][p] = c * a - s * b;
                    V[k][q] = s * a + c * b;
                }
            }
    }
    int order[MAXM];
    for (int i = 0; i < m; ++i) order[i] = i;
    std::sort(order, order + m, [&](int a, int b) { return C[a][a] < C[b][b]; });
    for (int jj = 0; jj < m; ++jj) {                          // S = L^-T V (back substitution per column), sorted
        const int j = order[jj];
        lam[jj] = C[j][j];
        for (int i = m - 1; i >= 0; --i) {
            double s = V[i][j];
            for (int k = i + 1; k < m; ++k) s -= L[k][i] * S[k * m + jj];
            S[i * m + jj] = s / L[i][i];
        }
    }
    return true;
}

}  // namespace

extern "C" int sem_fdm_setup(int64_t E, int m, const double* A, const double* B, double* S, double* inv_lambda) {
    if (E <= 0 || m < 2 || m > MAXM || !A || !B || !S || !inv_lambda) return SEM_EINVAL;
    const int64_t m2 = (int64_t)m * m, m3 = m2 * m;
    for (int64_t e = 0; e < E; ++e) {
        double lam[3][MAXM];
        for (int d = 0; d < 3; ++d)
            if (!gen_eig(m, A + (e * 3 + d) * m2, B + (e * 3 + d) * m2, S + (e * 3 + d) * m2, lam[d])) return SEM_EINVAL;
        double* il = inv_lambda + e * m3;
        for (int c = 0; c < m; ++c)
            for (int b = 0; b < m; ++b)
                for (int a = 0; a < m; ++a) il[(c * m + b) * m + a] = 1.0 / (lam[0][a] + lam[1][b] + lam[2][c]);
    }
    return SEM_OK;
}
