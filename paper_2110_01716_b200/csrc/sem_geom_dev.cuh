// sem_geom_dev.cuh — device helpers for the geometric factors (a2 / a9; P:69 isoparametric map; O3).
#pragma once

// 1-D tables handed to kernels by value (they land in the constant bank, so compile-time indices cost nothing).
struct Gll1D {
    double xi[16];
    double rho[16];
    double D[256];   // D[i*p + l]
};

// From the Jacobian Jm[a][b] = dx_a/dr_b and the quadrature weight W = rho_i rho_j rho_k:
//   G = (W / detJ) adj(Jm) adj(Jm)^T  (rr, rs, rt, ss, st, tt),  B = W detJ.   One division.  Returns detJ.
template <typename T>
__device__ __forceinline__ T sem_factors(const T (&J)[3][3], T W, T (&g)[6], T& B) {
    // rows of the adjugate: A_b = cofactor row so that R[b][a] = A[b][a] / det
    const T a00 = J[1][1] * J[2][2] - J[1][2] * J[2][1];
    const T a01 = J[0][2] * J[2][1] - J[0][1] * J[2][2];
    const T a02 = J[0][1] * J[1][2] - J[0][2] * J[1][1];
    const T a10 = J[1][2] * J[2][0] - J[1][0] * J[2][2];
    const T a11 = J[0][0] * J[2][2] - J[0][2] * J[2][0];
    const T a12 = J[0][2] * J[1][0] - J[0][0] * J[1][2];
    const T a20 = J[1][0] * J[2][1] - J[1][1] * J[2][0];
    const T a21 = J[0][1] * J[2][0] - J[0][0] * J[2][1];
    const T a22 = J[0][0] * J[1][1] - J[0][1] * J[1][0];
    const T det = J[0][0] * a00 + J[1][0] * a01 + J[2][0] * a02;
    const T s = W / det;
    g[0] = s * (a00 * a00 + a01 * a01 + a02 * a02);
    g[1] = s * (a00 * a10 + a01 * a11 + a02 * a12);
    g[2] = s * (a00 * a20 + a01 * a21 + a02 * a22);
    g[3] = s * (a10 * a10 + a11 * a11 + a12 * a12);
    g[4] = s * (a10 * a20 + a11 * a21 + a12 * a22);
    g[5] = s * (a20 * a20 + a21 * a21 + a22 * a22);
    B = W * det;
    return det;
}

// Jacobian of the trilinear blend of 8 vertices at (r,s,t) (S5).  X[v][d], v = a + 2b + 4c.
// x(r,s,t) = c0 + cr r + cs s + ct t + crs rs + crt rt + cst st + crst rst with the 8 coefficient vectors c*:
// the derivative is then 3 short polynomials.  coef[m][d], m = 0:1, 1:r, 2:s, 3:t, 4:rs, 5:rt, 6:st, 7:rst.
template <typename T>
__device__ __forceinline__ void sem_trilinear_coef(const T (&X)[8][3], T (&cf)[8][3]) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const T x0 = X[0][d], x1 = X[1][d], x2 = X[2][d], x3 = X[3][d], x4 = X[4][d], x5 = X[5][d], x6 = X[6][d],
                x7 = X[7][d];
        const T e = T(0.125);
        cf[0][d] = e * (((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7)));
        cf[1][d] = e * (((x1 - x0) + (x3 - x2)) + ((x5 - x4) + (x7 - x6)));
        cf[2][d] = e * (((x2 - x0) + (x3 - x1)) + ((x6 - x4) + (x7 - x5)));
        cf[3][d] = e * (((x4 - x0) + (x5 - x1)) + ((x6 - x2) + (x7 - x3)));
        cf[4][d] = e * (((x0 - x1) + (x3 - x2)) + ((x4 - x5) + (x7 - x6)));
        cf[5][d] = e * (((x0 - x1) + (x2 - x3)) + ((x5 - x4) + (x7 - x6)));
        cf[6][d] = e * (((x0 + x1) - (x2 + x3)) + ((x6 + x7) - (x4 + x5)));
        cf[7][d] = e * (((x1 - x0) + (x2 - x3)) + ((x4 - x5) + (x7 - x6)));
    }
}

template <typename T>
__device__ __forceinline__ void sem_trilinear_jac(const T (&cf)[8][3], T r, T s, T t, T (&J)[3][3]) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        J[d][0] = cf[1][d] + cf[4][d] * s + (cf[5][d] + cf[7][d] * s) * t;
        J[d][1] = cf[2][d] + cf[4][d] * r + (cf[6][d] + cf[7][d] * r) * t;
        J[d][2] = cf[3][d] + cf[5][d] * r + (cf[6][d] + cf[7][d] * r) * s;
    }
}
