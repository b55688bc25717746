// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU implementation of the spectral-element Poisson/Helmholtz hot path of
// arXiv 2110.01716 (Nek5000/RS), written from the paper's definitions (PAPER.md lines cited as P:nn) and the
// readings listed in DESIGN.md / SURVEY.md §8(c) (cited as O1..O8, S1..S22).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call this.
// It shares no code, header, table or constant with the CUDA path under paper_2110_01716_b200/csrc.
//
// Everything is `double`; dot products accumulate in `long double` so the oracle is the more accurate side.
// Parallelism: `#pragma omp parallel for` over elements / segments only (no blocking, fusion or reordering).
//
// Parity pins (tests/test_oracle_pins.py): closed-form GLL data, polynomial exactness of D, A*1 = 0, symmetry,
// volume, u=x energy, affine Kronecker form, dense brute-force assembly, exact diagonal, sin-product energy,
// spectral convergence, dense Cholesky solve, Krylov optimality, element-permutation invariance.
// Random-input outputs (e.g. ||w||_inf for a seeded u) are "parity unpinned" except through those structural pins.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// Legendre polynomial P_n(x) and P_{n-1}(x) by the three-term recurrence (textbook; Deville-Fischer-Mund).
inline void legendre(int n, long double x, long double& Pn, long double& Pnm1) {
    long double p0 = 1.0L, p1 = x;
    if (n == 0) { Pn = 1.0L; Pnm1 = 0.0L; return; }
    for (int m = 1; m < n; ++m) {
        long double p2 = ((2 * m + 1) * x * p1 - m * p0) / (m + 1);
        p0 = p1; p1 = p2;
    }
    Pn = p1; Pnm1 = p0;
}

inline int64_t p3_of(int N) { int64_t p = N + 1; return p * p * p; }

}  // namespace

extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// O1 ("Gauss-Lobatto-Legendre (GLL) quadrature points", "D_il := dh_l/dr at xi_i").
// xi[p], rho[p], D[p*p] row-major, row = evaluation point i, column = basis function l.
int orc_gll(int N, double* xi, double* rho, double* D) {
    if (N < 1) return -1;
    const int p = N + 1;
    std::vector<long double> x(p), PN(p);
    x[0] = -1.0L; x[N] = 1.0L;
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int i = 1; i < N; ++i) {
        long double xx = -std::cos(pi * i / N);          // Chebyshev-Lobatto initial guess
        for (int it = 0; it < 100; ++it) {
            long double Pn, Pm;
            legendre(N, xx, Pn, Pm);
            long double dP = N * (xx * Pn - Pm) / (xx * xx - 1.0L);                     // P_N'(x)
            long double d2P = (2.0L * xx * dP - (long double)N * (N + 1) * Pn) / (1.0L - xx * xx);  // P_N''(x)
            long double dx = dP / d2P;
            xx -= dx;
            if (std::fabs(dx) < 1e-19L) break;
        }
        x[i] = xx;
    }
    // enforce exact antisymmetry of the node set (it holds mathematically)
    for (int i = 0; i < p / 2; ++i) { long double a = 0.5L * (x[N - i] - x[i]); x[i] = -a; x[N - i] = a; }
    if (p % 2 == 1) x[N / 2] = 0.0L;
    for (int i = 0; i < p; ++i) {
        long double Pn, Pm;
        legendre(N, x[i], Pn, Pm);
        PN[i] = Pn;
        xi[i] = (double)x[i];
        rho[i] = (double)(2.0L / ((long double)N * (N + 1) * Pn * Pn));
    }
    for (int i = 0; i < p; ++i)
        for (int j = 0; j < p; ++j) {
            long double d;
            if (i != j) d = PN[i] / (PN[j] * (x[i] - x[j]));
            else if (i == 0) d = -(long double)N * (N + 1) / 4.0L;
            else if (i == N) d = (long double)N * (N + 1) / 4.0L;
            else d = 0.0L;
            D[i * p + j] = (double)d;
        }
    return 0;
}

// O2 (P:69 isoparametric map from [-1,1]^3; S5: elements are trilinear images of their 8 vertices).
// vert[E][8][3], vertex v = a + 2b + 4c sits at (r,s,t) = (2a-1, 2b-1, 2c-1); xyz[E][p^3][3], node l=(k*p+j)*p+i.
int orc_node_xyz(int64_t E, int N, const double* vert, double* xyz) {
    const int p = N + 1;
    std::vector<double> xi(p), rho(p), D(p * p);
    if (orc_gll(N, xi.data(), rho.data(), D.data())) return -1;
    const int64_t p3 = p3_of(N);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < E; ++e)
        for (int k = 0; k < p; ++k)
            for (int j = 0; j < p; ++j)
                for (int i = 0; i < p; ++i) {
                    const double r = xi[i], s = xi[j], t = xi[k];
                    double X[3] = {0, 0, 0};
                    for (int v = 0; v < 8; ++v) {
                        const int a = v & 1, b = (v >> 1) & 1, c = (v >> 2) & 1;
                        const double phi = 0.5 * (a ? 1 + r : 1 - r) * 0.5 * (b ? 1 + s : 1 - s) * 0.5 * (c ? 1 + t : 1 - t);
                        for (int d = 0; d < 3; ++d) X[d] += vert[(e * 8 + v) * 3 + d] * phi;
                    }
                    const int64_t l = ((int64_t)k * p + j) * p + i;
                    for (int d = 0; d < 3; ++d) xyz[(e * p3 + l) * 3 + d] = X[d];
                }
    return 0;
}

// Shared tail of O3: from the Jacobian matrix Jm[a][b] = dx_a/dr_b at one node and the weight W = rho_i rho_j rho_k,
// G_bc = W * detJ * sum_a R[b][a] R[c][a], R = Jm^{-1};  7th entry B = W * detJ.   Returns detJ.
static inline double factors_from_jacobian(const double Jm[3][3], double W, double g[7]) {
    const double det = Jm[0][0] * (Jm[1][1] * Jm[2][2] - Jm[1][2] * Jm[2][1])
                     - Jm[0][1] * (Jm[1][0] * Jm[2][2] - Jm[1][2] * Jm[2][0])
                     + Jm[0][2] * (Jm[1][0] * Jm[2][1] - Jm[1][1] * Jm[2][0]);
    double R[3][3];  // inverse by cofactors: R[b][a] = cof(Jm)[a][b] / det
    R[0][0] = (Jm[1][1] * Jm[2][2] - Jm[1][2] * Jm[2][1]) / det;
    R[0][1] = (Jm[0][2] * Jm[2][1] - Jm[0][1] * Jm[2][2]) / det;
    R[0][2] = (Jm[0][1] * Jm[1][2] - Jm[0][2] * Jm[1][1]) / det;
    R[1][0] = (Jm[1][2] * Jm[2][0] - Jm[1][0] * Jm[2][2]) / det;
    R[1][1] = (Jm[0][0] * Jm[2][2] - Jm[0][2] * Jm[2][0]) / det;
    R[1][2] = (Jm[0][2] * Jm[1][0] - Jm[0][0] * Jm[1][2]) / det;
    R[2][0] = (Jm[1][0] * Jm[2][1] - Jm[1][1] * Jm[2][0]) / det;
    R[2][1] = (Jm[0][1] * Jm[2][0] - Jm[0][0] * Jm[2][1]) / det;
    R[2][2] = (Jm[0][0] * Jm[1][1] - Jm[0][1] * Jm[1][0]) / det;
    auto dotrow = [&](int b, int c) { return R[b][0] * R[c][0] + R[b][1] * R[c][1] + R[b][2] * R[c][2]; };
    const double s = W * det;
    g[0] = s * dotrow(0, 0);  // G_rr
    g[1] = s * dotrow(0, 1);  // G_rs
    g[2] = s * dotrow(0, 2);  // G_rt
    g[3] = s * dotrow(1, 1);  // G_ss
    g[4] = s * dotrow(1, 2);  // G_st
    g[5] = s * dotrow(2, 2);  // G_tt
    g[6] = s;                 // B (diagonal mass)
    return det;
}

// O3, isoparametric route: Jm by applying D to the node coordinates in each direction.
// xyz[E][p^3][3] -> G[E][7][p^3] (rr,rs,rt,ss,st,tt,B), detJ[E][p^3].  Returns 0, or -2 if any detJ <= 0.
int orc_geom_iso(int64_t E, int N, const double* xyz, double* G, double* detJ) {
    const int p = N + 1;
    std::vector<double> xi(p), rho(p), D(p * p);
    if (orc_gll(N, xi.data(), rho.data(), D.data())) return -1;
    const int64_t p3 = p3_of(N);
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (int64_t e = 0; e < E; ++e) {
        const double* X = xyz + e * p3 * 3;
        for (int k = 0; k < p; ++k)
            for (int j = 0; j < p; ++j)
                for (int i = 0; i < p; ++i) {
                    double Jm[3][3];
                    for (int a = 0; a < 3; ++a) {
                        double dr = 0, ds = 0, dt = 0;
                        for (int l = 0; l < p; ++l) {
                            dr += D[i * p + l] * X[(((int64_t)k * p + j) * p + l) * 3 + a];
                            ds += D[j * p + l] * X[(((int64_t)k * p + l) * p + i) * 3 + a];
                            dt += D[k * p + l] * X[(((int64_t)l * p + j) * p + i) * 3 + a];
                        }
                        Jm[a][0] = dr; Jm[a][1] = ds; Jm[a][2] = dt;
                    }
                    double g[7];
                    const double det = factors_from_jacobian(Jm, rho[i] * rho[j] * rho[k], g);
                    if (!(det > 0)) bad |= 1;
                    const int64_t l = ((int64_t)k * p + j) * p + i;
                    for (int c = 0; c < 7; ++c) G[(e * 7 + c) * p3 + l] = g[c];
                    detJ[e * p3 + l] = det;
                }
    }
    return bad ? -2 : 0;
}

// O3, trilinear-analytic route (S5; the recomputed-G variant a9): Jm from the derivative of the trilinear blend.
int orc_geom_trilinear(int64_t E, int N, const double* vert, double* G, double* detJ) {
    const int p = N + 1;
    std::vector<double> xi(p), rho(p), D(p * p);
    if (orc_gll(N, xi.data(), rho.data(), D.data())) return -1;
    const int64_t p3 = p3_of(N);
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (int64_t e = 0; e < E; ++e)
        for (int k = 0; k < p; ++k)
            for (int j = 0; j < p; ++j)
                for (int i = 0; i < p; ++i) {
                    const double r = xi[i], s = xi[j], t = xi[k];
                    double Jm[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
                    for (int v = 0; v < 8; ++v) {
                        const int a = v & 1, b = (v >> 1) & 1, c = (v >> 2) & 1;
                        const double fr = 0.5 * (a ? 1 + r : 1 - r), fs = 0.5 * (b ? 1 + s : 1 - s), ft = 0.5 * (c ? 1 + t : 1 - t);
                        const double dfr = a ? 0.5 : -0.5, dfs = b ? 0.5 : -0.5, dft = c ? 0.5 : -0.5;
                        for (int d = 0; d < 3; ++d) {
                            const double Xv = vert[(e * 8 + v) * 3 + d];
                            Jm[d][0] += Xv * dfr * fs * ft;
                            Jm[d][1] += Xv * fr * dfs * ft;
                            Jm[d][2] += Xv * fr * fs * dft;
                        }
                    }
                    double g[7];
                    const double det = factors_from_jacobian(Jm, rho[i] * rho[j] * rho[k], g);
                    if (!(det > 0)) bad |= 1;
                    const int64_t l = ((int64_t)k * p + j) * p + i;
                    for (int c = 0; c < 7; ++c) G[(e * 7 + c) * p3 + l] = g[c];
                    detJ[e * p3 + l] = det;
                }
    return bad ? -2 : 0;
}

// O4 (P:93 for the contraction u_r,ijk = sum_l D_il u_ljk; "A is the discrete equivalent of -laplacian, SPD";
// S1/S2: the GLL-collocated weak Laplacian).  Local operator w = D^T G D u (+ lambda B u), element by element, no gs.
// u[E][p^3], G[E][7][p^3], w[E][p^3].
int orc_ax(int64_t E, int N, const double* G, const double* u, double* w, double lambda) {
    const int p = N + 1;
    std::vector<double> xi(p), rho(p), D(p * p);
    if (orc_gll(N, xi.data(), rho.data(), D.data())) return -1;
    const int64_t p3 = p3_of(N);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < E; ++e) {
        const double* ue = u + e * p3;
        const double* Ge = G + e * 7 * p3;
        double* we = w + e * p3;
        std::vector<double> gr(p3), gs(p3), gt(p3);
        auto at = [p](int k, int j, int i) { return ((int64_t)k * p + j) * p + i; };
        for (int k = 0; k < p; ++k)
            for (int j = 0; j < p; ++j)
                for (int i = 0; i < p; ++i) {
                    double ur = 0, us = 0, ut = 0;
                    for (int l = 0; l < p; ++l) {
                        ur += D[i * p + l] * ue[at(k, j, l)];
                        us += D[j * p + l] * ue[at(k, l, i)];
                        ut += D[k * p + l] * ue[at(l, j, i)];
                    }
                    const int64_t n = at(k, j, i);
                    const double Grr = Ge[0 * p3 + n], Grs = Ge[1 * p3 + n], Grt = Ge[2 * p3 + n];
                    const double Gss = Ge[3 * p3 + n], Gst = Ge[4 * p3 + n], Gtt = Ge[5 * p3 + n];
                    gr[n] = Grr * ur + Grs * us + Grt * ut;
                    gs[n] = Grs * ur + Gss * us + Gst * ut;
                    gt[n] = Grt * ur + Gst * us + Gtt * ut;
                }
        for (int k = 0; k < p; ++k)
            for (int j = 0; j < p; ++j)
                for (int i = 0; i < p; ++i) {
                    double acc = 0;
                    for (int l = 0; l < p; ++l) {
                        acc += D[l * p + i] * gr[at(k, j, l)];
                        acc += D[l * p + j] * gs[at(k, l, i)];
                        acc += D[l * p + k] * gt[at(l, j, i)];
                    }
                    const int64_t n = at(k, j, i);
                    if (lambda != 0.0) acc += lambda * Ge[6 * p3 + n] * ue[n];
                    we[n] = acc;
                }
    }
    return 0;
}

// O6 ("the user simply provides a global ID for each vertex"): canonical maps from gid[nL].
// Pass 1: number of distinct gids.
int64_t orc_count_unique(int64_t nL, const int64_t* gid) {
    std::vector<int64_t> s(gid, gid + nL);
    std::sort(s.begin(), s.end());
    return (int64_t)(std::unique(s.begin(), s.end()) - s.begin());
}

// Pass 2: uniq_gid[U] ascending; l2u[nL] = rank of gid[l]; mult[U]; seg_off[U+1] = exclusive scan of mult;
// seg_idx[nL] = local indices ordered by (l2u, l) ascending (a stable sort of l by gid).
int orc_maps(int64_t nL, const int64_t* gid, int64_t U, int64_t* uniq_gid, int32_t* l2u, int32_t* mult,
             int64_t* seg_off, int32_t* seg_idx) {
    for (int64_t l = 0; l < nL; ++l) if (gid[l] < 0) return -1;
    std::vector<int64_t> order(nL);
    std::iota(order.begin(), order.end(), (int64_t)0);
    std::stable_sort(order.begin(), order.end(), [gid](int64_t a, int64_t b) { return gid[a] < gid[b]; });
    int64_t g = -1;
    int64_t prev = -1;
    for (int64_t q = 0; q < nL; ++q) {
        const int64_t l = order[q];
        if (q == 0 || gid[l] != prev) {
            ++g;
            if (g >= U) return -1;
            uniq_gid[g] = gid[l];
            mult[g] = 0;
            seg_off[g] = q;
            prev = gid[l];
        }
        l2u[l] = (int32_t)g;
        mult[g] += 1;
        seg_idx[q] = (int32_t)l;
    }
    if (g + 1 != U) return -1;
    seg_off[U] = nL;
    return 0;
}

// O5 ("exchange-and-sum of shared interface values"): s[g] = sum over copies in ascending l; w[l] = s[l2u[l]].
int orc_gs(int64_t nL, int64_t U, const int32_t* l2u, double* w) {
    std::vector<double> s(U, 0.0);
    for (int64_t l = 0; l < nL; ++l) s[l2u[l]] += w[l];
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < nL; ++l) w[l] = s[l2u[l]];
    return 0;
}

// O7 / S12: exact diagonal of the local operator (including the cross terms that survive at element ends).
int orc_diag_local(int64_t E, int N, const double* G, double* diag, double lambda) {
    const int p = N + 1;
    std::vector<double> xi(p), rho(p), D(p * p);
    if (orc_gll(N, xi.data(), rho.data(), D.data())) return -1;
    const int64_t p3 = p3_of(N);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < E; ++e) {
        const double* Ge = G + e * 7 * p3;
        auto at = [p](int k, int j, int i) { return ((int64_t)k * p + j) * p + i; };
        for (int k = 0; k < p; ++k)
            for (int j = 0; j < p; ++j)
                for (int i = 0; i < p; ++i) {
                    double d = 0;
                    for (int l = 0; l < p; ++l) {
                        d += D[l * p + i] * D[l * p + i] * Ge[0 * p3 + at(k, j, l)];
                        d += D[l * p + j] * D[l * p + j] * Ge[3 * p3 + at(k, l, i)];
                        d += D[l * p + k] * D[l * p + k] * Ge[5 * p3 + at(l, j, i)];
                    }
                    const int64_t n = at(k, j, i);
                    d += 2.0 * (D[i * p + i] * D[j * p + j] * Ge[1 * p3 + n] + D[i * p + i] * D[k * p + k] * Ge[2 * p3 + n]
                                + D[j * p + j] * D[k * p + k] * Ge[4 * p3 + n]);
                    if (lambda != 0.0) d += lambda * Ge[6 * p3 + n];
                    diag[e * p3 + n] = d;
                }
    }
    return 0;
}

// Masked assembled operator in unique-node storage (O8, S14): y = M Q^T A_L Q M x.
// mask_u[U]: 1 = Dirichlet (masked) node.  Scratch uL, wL of size nL supplied by the caller.
static void apply_Ag(int64_t E, int N, const double* G, double lambda, int64_t nL, int64_t U, const int32_t* l2u,
                     const uint8_t* mask_u, const double* x, double* y, double* uL, double* wL) {
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < nL; ++l) { const int32_t g = l2u[l]; uL[l] = mask_u[g] ? 0.0 : x[g]; }
    orc_ax(E, N, G, uL, wL, lambda);
    for (int64_t g = 0; g < U; ++g) y[g] = 0.0;
    for (int64_t l = 0; l < nL; ++l) y[l2u[l]] += wL[l];
    for (int64_t g = 0; g < U; ++g) if (mask_u[g]) y[g] = 0.0;
}

int orc_apply_Ag(int64_t E, int N, const double* G, double lambda, int64_t nL, int64_t U, const int32_t* l2u,
                 const uint8_t* mask_u, const double* x, double* y) {
    std::vector<double> uL(nL), wL(nL);
    apply_Ag(E, N, G, lambda, nL, U, l2u, mask_u, x, y, uL.data(), wL.data());
    return 0;
}

static long double dotL(int64_t n, const double* a, const double* b) {
    long double s = 0.0L;
    for (int64_t i = 0; i < n; ++i) s += (long double)a[i] * (long double)b[i];
    return s;
}

// O8 ("Jacobi-preconditioned conjugate gradient iteration"; S13 stopping rule; S12 exact diagonal).
// All vectors in unique storage.  b must be assembled and zero at masked nodes.  x: in x0, out solution.
// relres_hist[maxit+1]: ||r||/||r0|| after each iteration (entry 0 = 1).  snap_its[ns] ascending iteration numbers
// at which x is copied to x_snap[ns][U] (nullable).  Returns iterations done (operator applications in the loop).
int orc_pcg(int64_t E, int N, const double* G, double lambda, int64_t nL, int64_t U, const int32_t* l2u,
            const uint8_t* mask_u, const double* b, double* x, double tol, int maxit, double* relres_out,
            double* relres_hist, int ns, const int* snap_its, double* x_snap) {
    std::vector<double> uL(nL), wL(nL), diagL(nL), Minv(U, 0.0), r(U), z(U), pv(U), q(U);
    orc_diag_local(E, N, G, diagL.data(), lambda);
    {
        std::vector<double> dg(U, 0.0);
        for (int64_t l = 0; l < nL; ++l) dg[l2u[l]] += diagL[l];
        for (int64_t g = 0; g < U; ++g) Minv[g] = mask_u[g] ? 0.0 : 1.0 / dg[g];
    }
    for (int64_t g = 0; g < U; ++g) if (mask_u[g]) x[g] = 0.0;
    bool x0zero = true;
    for (int64_t g = 0; g < U; ++g) if (x[g] != 0.0) { x0zero = false; break; }
    if (x0zero) { for (int64_t g = 0; g < U; ++g) r[g] = mask_u[g] ? 0.0 : b[g]; }
    else {
        apply_Ag(E, N, G, lambda, nL, U, l2u, mask_u, x, q.data(), uL.data(), wL.data());
        for (int64_t g = 0; g < U; ++g) r[g] = mask_u[g] ? 0.0 : b[g] - q[g];
    }
    for (int64_t g = 0; g < U; ++g) { z[g] = Minv[g] * r[g]; pv[g] = z[g]; }
    long double rho = dotL(U, r.data(), z.data());
    const long double r0 = std::sqrt(dotL(U, r.data(), r.data()));
    if (relres_hist) relres_hist[0] = 1.0;
    if (relres_out) *relres_out = (r0 == 0.0L) ? 0.0 : 1.0;
    if (r0 == 0.0L) return 0;
    int it = 0, snap = 0;
    while (it < maxit) {
        ++it;
        apply_Ag(E, N, G, lambda, nL, U, l2u, mask_u, pv.data(), q.data(), uL.data(), wL.data());
        const long double pq = dotL(U, pv.data(), q.data());
        if (!(pq > 0.0L)) { if (relres_hist) relres_hist[it] = relres_hist[it - 1]; break; }  // breakdown (S13)
        const double alpha = (double)(rho / pq);
        for (int64_t g = 0; g < U; ++g) { x[g] += alpha * pv[g]; r[g] -= alpha * q[g]; }
        const long double rr = std::sqrt(dotL(U, r.data(), r.data()));
        const double rel = (double)(rr / r0);
        if (relres_hist) relres_hist[it] = rel;
        if (relres_out) *relres_out = rel;
        while (snap < ns && snap_its[snap] == it) { std::memcpy(x_snap + (int64_t)snap * U, x, sizeof(double) * U); ++snap; }
        if (rr <= (long double)tol * r0) break;
        for (int64_t g = 0; g < U; ++g) z[g] = Minv[g] * r[g];
        const long double rho2 = dotL(U, r.data(), z.data());
        const double beta = (double)(rho2 / rho);
        rho = rho2;
        for (int64_t g = 0; g < U; ++g) pv[g] = z[g] + beta * pv[g];
    }
    return it;
}

// ---- NEXT-1: p-multigrid transfer operators ----------------------------------------------------
// P:103 "Coarse-to-fine interpolations are cast as efficient tensor contractions, u_f = (J x J x J) u_c, where J is the
// 1D polynomial interpolation operator from the coarse GLL points to the fine GLL points."
// J[i*(Nc+1) + j] = h^c_j(xi^f_i): Lagrange cardinal function j of the Nc+1 coarse GLL points at fine GLL point i,
// written out as the plain product formula  prod_{m != j} (x - xi^c_m) / (xi^c_j - xi^c_m).
int orc_interp(int Nc, int Nf, double* J) {
    if (Nc < 1 || Nf < 1) return -1;
    const int pc = Nc + 1, pf = Nf + 1;
    std::vector<double> xc(pc), xf(pf), rho(std::max(pc, pf)), D((size_t)std::max(pc, pf) * std::max(pc, pf));
    orc_gll(Nc, xc.data(), rho.data(), D.data());
    orc_gll(Nf, xf.data(), rho.data(), D.data());
    for (int i = 0; i < pf; ++i)
        for (int j = 0; j < pc; ++j) {
            long double h = 1.0L;
            for (int m = 0; m < pc; ++m)
                if (m != j) h *= ((long double)xf[i] - (long double)xc[m]) / ((long double)xc[j] - (long double)xc[m]);
            J[i * pc + j] = (double)h;
        }
    return 0;
}

// Prolongation, element by element (local layout, i fastest):  uf[k][j][i] = sum_{c,b,a} J[k][c] J[j][b] J[i][a] uc[c][b][a].
int orc_prolong(int64_t E, int Nc, int Nf, const double* uc, double* uf) {
    const int pc = Nc + 1, pf = Nf + 1;
    std::vector<double> J((size_t)pf * pc);
    if (orc_interp(Nc, Nf, J.data())) return -1;
    const int64_t pc3 = (int64_t)pc * pc * pc, pf3 = (int64_t)pf * pf * pf;
#pragma omp parallel for
    for (int64_t e = 0; e < E; ++e)
        for (int k = 0; k < pf; ++k)
            for (int j = 0; j < pf; ++j)
                for (int i = 0; i < pf; ++i) {
                    long double s = 0.0L;
                    for (int c = 0; c < pc; ++c)
                        for (int b = 0; b < pc; ++b)
                            for (int a = 0; a < pc; ++a)
                                s += (long double)J[k * pc + c] * J[j * pc + b] * J[i * pc + a] *
                                     uc[e * pc3 + ((int64_t)c * pc + b) * pc + a];
                    uf[e * pf3 + ((int64_t)k * pf + j) * pf + i] = (double)s;
                }
    return 0;
}

// Restriction = the transpose of the prolongation (residuals are functionals: r_c = (J^T x J^T x J^T) r_f), element by
// element:  rc[c][b][a] = sum_{k,j,i} J[k][c] J[j][b] J[i][a] rf[k][j][i].
int orc_restrict(int64_t E, int Nc, int Nf, const double* rf, double* rc) {
    const int pc = Nc + 1, pf = Nf + 1;
    std::vector<double> J((size_t)pf * pc);
    if (orc_interp(Nc, Nf, J.data())) return -1;
    const int64_t pc3 = (int64_t)pc * pc * pc, pf3 = (int64_t)pf * pf * pf;
#pragma omp parallel for
    for (int64_t e = 0; e < E; ++e)
        for (int c = 0; c < pc; ++c)
            for (int b = 0; b < pc; ++b)
                for (int a = 0; a < pc; ++a) {
                    long double s = 0.0L;
                    for (int k = 0; k < pf; ++k)
                        for (int j = 0; j < pf; ++j)
                            for (int i = 0; i < pf; ++i)
                                s += (long double)J[k * pc + c] * J[j * pc + b] * J[i * pc + a] *
                                     rf[e * pf3 + ((int64_t)k * pf + j) * pf + i];
                    rc[e * pc3 + ((int64_t)c * pc + b) * pc + a] = (double)s;
                }
    return 0;
}

// ---- NEXT-1: Chebyshev-accelerated point-Jacobi smoother ("Smoothers for pMG include Chebyshev-accelerated
// point-Jacobi") ---------------------------------------------------------------------------------------------------
// The paper names the smoother and nothing else (reading S23): this is the textbook Chebyshev semi-iteration
// (Saad, Iterative Methods, Alg. 12.1) on the Jacobi-preconditioned operator M^-1 A with M = diag(A), for eigenvalue
// bounds [lmin, lmax] of M^-1 A supplied by the caller:
//   theta = (lmax+lmin)/2, delta = (lmax-lmin)/2, sigma = theta/delta, rho_0 = 1/sigma
//   r = M^-1 (b - A x);  d = r / theta
//   for k = 1 .. order-1:  x += d;  r -= M^-1 A d;  rho_k = 1/(2 sigma - rho_{k-1});
//                          d = rho_k rho_{k-1} d + (2 rho_k / delta) r
//   x += d
// so `order` applications of M^-1 are made and the error is multiplied by T_order((theta - t)/delta)/T_order(sigma) on
// the eigenvalue t of M^-1 A.  Unique storage; A = masked assembled operator (O8), b assembled and masked.
int orc_cheby(int64_t E, int N, const double* G, double lambda, int64_t nL, int64_t U, const int32_t* l2u,
              const uint8_t* mask_u, const double* b, double* x, int order, double lmin, double lmax) {
    if (order < 1 || !(lmax > lmin) || !(lmin > 0.0)) return -1;
    std::vector<double> uL(nL), wL(nL), diagL(nL), Minv(U, 0.0), r(U), d(U), q(U);
    orc_diag_local(E, N, G, diagL.data(), lambda);
    {
        std::vector<double> dg(U, 0.0);
        for (int64_t l = 0; l < nL; ++l) dg[l2u[l]] += diagL[l];
        for (int64_t g = 0; g < U; ++g) Minv[g] = mask_u[g] ? 0.0 : 1.0 / dg[g];
    }
    const double theta = 0.5 * (lmax + lmin), delta = 0.5 * (lmax - lmin), sigma = theta / delta;
    double rho = 1.0 / sigma;
    for (int64_t g = 0; g < U; ++g) if (mask_u[g]) x[g] = 0.0;
    apply_Ag(E, N, G, lambda, nL, U, l2u, mask_u, x, q.data(), uL.data(), wL.data());
    for (int64_t g = 0; g < U; ++g) { r[g] = Minv[g] * (b[g] - q[g]); d[g] = r[g] / theta; }
    for (int k = 1; k < order; ++k) {
        for (int64_t g = 0; g < U; ++g) x[g] += d[g];
        apply_Ag(E, N, G, lambda, nL, U, l2u, mask_u, d.data(), q.data(), uL.data(), wL.data());
        const double rho1 = 1.0 / (2.0 * sigma - rho);
        for (int64_t g = 0; g < U; ++g) {
            r[g] -= Minv[g] * q[g];
            d[g] = rho1 * rho * d[g] + (2.0 * rho1 / delta) * r[g];
        }
        rho = rho1;
    }
    for (int64_t g = 0; g < U; ++g) x[g] += d[g];
    return 0;
}

}  // extern "C"
