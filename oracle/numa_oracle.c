/*
 * numa_oracle.c -- CPU FP64 ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct restatement of the hot path of arXiv 2504.08157
 * (xNUMA): the matrix-free continuous-Galerkin spectral-element right-hand side of the
 * compressible Euler equations in perturbation form q = (rho', u, v, w, theta')
 * (Eq. 1-3), its global assembly (Eq. 10-12, Alg. 3) and the explicit
 * Runge-Kutta stage update that consumes it.  Every function cites the passage it follows.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may build, load or call this file.  It shares NO code, header, table or constant
 * generator with the CUDA path (paper_2504_08157_b200/csrc); neither includes the other.
 *
 * No blocking, fusion, vectorisation or reordering beyond what the paper's algorithms
 * state.  OpenMP only distributes whole elements (or whole fields) across threads; the
 * arithmetic per element is the plain nested loop of Alg. 2.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): LGL closed forms, quadrature exactness,
 * polynomial exactness of D and of the metric/gradient on deformed meshes, volume
 * identity sum(wJ) = |Omega|, free stream, atmosphere at rest (bitwise zero), buoyancy
 * closed form, global mass conservation, DSS projection algebra vs an explicit Q Q^T,
 * manufactured-solution convergence order, RK3 amplification polynomial, linear
 * acoustics speed, wall projection, and a NumPy Kronecker brute-force restatement (P1-P16);
 * orc_sources: Coriolis turns the wind clockwise by f t and conserves its speed, the sponge
 * decays as exp(-beta t) and leaves rho' alone, heating raises theta' only (P17-P19);
 * RI diagnostic (P20-P25), hyper-diffusion (P26-P31), IMEX linear operator / ARK2 / GMRES
 * (P32-P36), the u . grad theta0 term of Eq. 1c and the L_theta row of the linear operator in
 * closed form on the constant-N_BV sounding (P37) -- see the test files named at each function.
 * Physical fidelity of the tropical-cyclone run itself is "parity unpinned" (the observed
 * heating data of PAPER.md:L312 is not available).
 *
 * Layout (q_e(i,j,k,e,m)): field[m][e][n], n = i + Nq*(j + Nq*k).
 * met[3*a + c][e][n] = d xi_a / d x_c  (a: xi,eta,zeta; c: x,y,z).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define NODE(i, j, k) ((i) + Nq * ((j) + Nq * (k)))

/* ------------------------------------------------------------------------------------
 * A0.1  LGL points, weights, derivative matrix.
 * PAPER.md:L88 (Eq. 5: Lagrange polynomials at the LGL points), L103-L109 (Eq. 8:
 * quadrature weights at the LGL points).  Closed forms (textbook): points are +-1 and the
 * roots of P'_N; w_i = 2 / (N (N+1) P_N(xi_i)^2).
 * ---------------------------------------------------------------------------------- */
static void legendre(int N, double x, double *P, double *dP, double *d2P)
{
    /* Bonnet recurrence (n+1) P_{n+1} = (2n+1) x P_n - n P_{n-1} */
    double p0 = 1.0, p1 = x;
    if (N == 0) { *P = 1.0; *dP = 0.0; *d2P = 0.0; return; }
    for (int n = 1; n < N; ++n) {
        double p2 = ((2.0 * n + 1.0) * x * p1 - n * p0) / (n + 1.0);
        p0 = p1; p1 = p2;
    }
    *P = p1;
    /* (1-x^2) P'_N = N (P_{N-1} - x P_N);  Legendre ODE gives P''_N */
    double om = 1.0 - x * x;
    *dP = N * (p0 - x * p1) / om;
    *d2P = (2.0 * x * (*dP) - N * (N + 1.0) * p1) / om;
}

void orc_lgl(int N, double *xi, double *w)
{
    const double pi = 3.14159265358979323846;
    xi[0] = -1.0; xi[N] = 1.0;
    for (int i = 1; i < N; ++i) {
        double x = -cos(pi * i / N); /* Chebyshev-Gauss-Lobatto initial guess */
        for (int it = 0; it < 100; ++it) {
            double P, dP, d2P;
            legendre(N, x, &P, &dP, &d2P);
            double dx = dP / d2P;
            x -= dx;
            if (fabs(dx) < 1e-16) break;
        }
        xi[i] = x;
    }
    for (int i = 0; i <= N; ++i) {
        double P, dP, d2P;
        if (i == 0 || i == N) {
            /* P_N(+-1) = (+-1)^N */
            P = (i == N || N % 2 == 0) ? 1.0 : -1.0;
        } else {
            legendre(N, xi[i], &P, &dP, &d2P);
        }
        w[i] = 2.0 / (N * (N + 1.0) * P * P);
    }
}

/* D[i*Nq + l] = h'_l(xi_i): derivative of the l-th Lagrange polynomial at point i.
 * The paper's d phi/d xi (l, i) (Alg. 2) is D[i][l] (Q5).
 * h'_l(xi_i) = P_N(xi_i) / (P_N(xi_l) (xi_i - xi_l)), i != l; diagonal = -(row sum). */
void orc_dmat(int N, const double *xi, double *D)
{
    int Nq = N + 1;
    double PN[64];
    for (int i = 0; i < Nq; ++i) {
        double dP, d2P;
        if (i == 0) PN[i] = (N % 2 == 0) ? 1.0 : -1.0;
        else if (i == N) PN[i] = 1.0;
        else legendre(N, xi[i], &PN[i], &dP, &d2P);
    }
    for (int i = 0; i < Nq; ++i) {
        double rowsum = 0.0;
        for (int l = 0; l < Nq; ++l) {
            if (l == i) continue;
            D[i * Nq + l] = PN[i] / (PN[l] * (xi[i] - xi[l]));
            rowsum += D[i * Nq + l];
        }
        D[i * Nq + i] = -rowsum;
    }
}

/* ------------------------------------------------------------------------------------
 * Alg. 2: reference-space derivatives of one nodal field on one
 * element:  f_xi(i,j,k) = sum_l D[i][l] f(l,j,k), f_eta = sum_l D[j][l] f(i,l,k),
 * f_zeta = sum_l D[k][l] f(i,j,l).  hold1/2/3 of the listing are fx/fe/fz.
 * ---------------------------------------------------------------------------------- */
static void ref_derivs_abs(int Nq, const double *D, const double *f, int i, int j, int k,
                           double *fx, double *fe, double *fz)
{
    double a1 = 0.0, a2 = 0.0, a3 = 0.0;
    for (int l = 0; l < Nq; ++l) {
        a1 += fabs(D[i * Nq + l] * f[NODE(l, j, k)]);
        a2 += fabs(D[j * Nq + l] * f[NODE(i, l, k)]);
        a3 += fabs(D[k * Nq + l] * f[NODE(i, j, l)]);
    }
    *fx = a1; *fe = a2; *fz = a3;
}

static void ref_derivs(int Nq, const double *D, const double *f, int i, int j, int k,
                       double *fx, double *fe, double *fz)
{
    double hold1 = 0.0, hold2 = 0.0, hold3 = 0.0;
    for (int l = 0; l < Nq; ++l) {
        hold1 = hold1 + D[i * Nq + l] * f[NODE(l, j, k)];
        hold2 = hold2 + D[j * Nq + l] * f[NODE(i, l, k)];
        hold3 = hold3 + D[k * Nq + l] * f[NODE(i, j, l)];
    }
    *fx = hold1; *fe = hold2; *fz = hold3;
}

/* Alg. 2 in difference form (see orc_metrics): sum_{l != i} D[i][l] (f_l - f_i). */
static void ref_derivs_diff(int Nq, const double *D, const double *f, int i, int j, int k,
                            double *fx, double *fe, double *fz)
{
    double hold1 = 0.0, hold2 = 0.0, hold3 = 0.0, f0 = f[NODE(i, j, k)];
    for (int l = 0; l < Nq; ++l) {
        if (l != i) hold1 = hold1 + D[i * Nq + l] * (f[NODE(l, j, k)] - f0);
        if (l != j) hold2 = hold2 + D[j * Nq + l] * (f[NODE(i, l, k)] - f0);
        if (l != k) hold3 = hold3 + D[k * Nq + l] * (f[NODE(i, j, l)] - f0);
    }
    *fx = hold1; *fe = hold2; *fz = hold3;
}

/* ------------------------------------------------------------------------------------
 * A0.2  Metric terms ("mapped ... via metric terms", L149 J = dx/dxi of the
 * isoparametric mapping; formula per DESIGN.md Q4): differentiate the nodal coordinates
 * with D, J = det(dx/dxi), grad xi_a = rows of the inverse (cross products / J).
 * The coordinate derivatives are evaluated in difference form,
 *   x_xi(i,j,k) = sum_{l != i} D[i][l] (x(l,j,k) - x(i,j,k)),
 * which is Alg. 2's sum with the diagonal entry D[i][i] = -sum_{l != i} D[i][l] written out
 * (identical in exact arithmetic).  A coordinate that is constant along a reference
 * direction then has an exactly zero derivative, and the round-off is relative to the
 * element size instead of to the distance from the origin (Q4).
 * Returns the number of nodes with J <= 0.
 * ---------------------------------------------------------------------------------- */
long orc_metrics(int N, long Ne, const double *xyz, double *met, double *jac)
{
    int Nq = N + 1;
    long Mn = (long)Nq * Nq * Nq, NL = Ne * Mn;
    double xi[64], w[64], D[64 * 64];
    orc_lgl(N, xi, w);
    orc_dmat(N, xi, D);
    long bad = 0;
#pragma omp parallel for reduction(+ : bad) schedule(static)
    for (long e = 0; e < Ne; ++e) {
        const double *x = xyz + 0 * NL + e * Mn, *y = xyz + 1 * NL + e * Mn, *z = xyz + 2 * NL + e * Mn;
        for (int k = 0; k < Nq; ++k)
            for (int j = 0; j < Nq; ++j)
                for (int i = 0; i < Nq; ++i) {
                    double xx, xe, xz, yx, ye, yz, zx, ze, zz;
                    ref_derivs_diff(Nq, D, x, i, j, k, &xx, &xe, &xz);
                    ref_derivs_diff(Nq, D, y, i, j, k, &yx, &ye, &yz);
                    ref_derivs_diff(Nq, D, z, i, j, k, &zx, &ze, &zz);
                    /* J = x_xi . (x_eta x x_zeta) */
                    double c0 = ye * zz - yz * ze, c1 = xz * ze - xe * zz, c2 = xe * yz - xz * ye;
                    double J = xx * c0 + yx * c1 + zx * c2;
                    long p = e * Mn + NODE(i, j, k);
                    jac[p] = J;
                    if (!(J > 0.0)) bad++;
                    /* grad xi = (x_eta x x_zeta)/J */
                    met[0 * NL + p] = c0 / J;
                    met[1 * NL + p] = c1 / J;
                    met[2 * NL + p] = c2 / J;
                    /* grad eta = (x_zeta x x_xi)/J */
                    met[3 * NL + p] = (yz * zx - yx * zz) / J;
                    met[4 * NL + p] = (xx * zz - xz * zx) / J;
                    met[5 * NL + p] = (xz * yx - xx * yz) / J;
                    /* grad zeta = (x_xi x x_eta)/J */
                    met[6 * NL + p] = (yx * ze - ye * zx) / J;
                    met[7 * NL + p] = (xe * zx - xx * ze) / J;
                    met[8 * NL + p] = (xx * ye - xe * yx) / J;
                }
    }
    return bad;
}

/* ------------------------------------------------------------------------------------
 * A0.3  Quadrature weight times Jacobian, diagonal mass, assembly weight.
 * PAPER.md Eq. 8 (L107): wJ = w_i w_j w_k J_ijk.  Eq. 10 with collocated (inexact)
 * integration (L117-L121): M_I = sum over local copies (e,ijk)->I of wJ.
 * omega = wJ / M_I is the factor that turns the local tendency S into the local
 * contribution to M^-1 R (Eq. 11-12; Q3).
 * ---------------------------------------------------------------------------------- */
void orc_mass(int N, long Ne, long NG, const int32_t *intma_cg, const double *jac,
              double *wJ, double *M, double *omega)
{
    int Nq = N + 1;
    long Mn = (long)Nq * Nq * Nq, NL = Ne * Mn;
    double xi[64], w[64];
    orc_lgl(N, xi, w);
    for (long e = 0; e < Ne; ++e)
        for (int k = 0; k < Nq; ++k)
            for (int j = 0; j < Nq; ++j)
                for (int i = 0; i < Nq; ++i) {
                    long p = e * Mn + NODE(i, j, k);
                    wJ[p] = w[i] * w[j] * w[k] * jac[p];
                }
    for (long I = 0; I < NG; ++I) M[I] = 0.0;
    for (long p = 0; p < NL; ++p) M[intma_cg[p]] += wJ[p];
    for (long p = 0; p < NL; ++p) omega[p] = wJ[p] / M[intma_cg[p]];
}

/* ------------------------------------------------------------------------------------
 * A0.4  No-flux wall entries ("a no-flux boundary condition is enforced";
 * implementation per DESIGN.md Q8): for every element face flagged as wall, one entry
 * (local node, outward unit normal) per face node; the outward normal of face
 * xi_a = -+1 is -+ grad xi_a / |grad xi_a|.  Entries are listed in (e, face, node) order.
 * Call with node == NULL to count.
 * ---------------------------------------------------------------------------------- */
long orc_wall_list(int N, long Ne, const uint8_t *face_bc, const double *met,
                   int64_t *node, double *normal /* [count][3] */)
{
    int Nq = N + 1;
    long Mn = (long)Nq * Nq * Nq, NL = Ne * Mn;
    long cnt = 0;
    for (long e = 0; e < Ne; ++e)
        for (int f = 0; f < 6; ++f) {
            if (!face_bc[e * 6 + f]) continue;
            int a = f / 2;
            double sgn = (f % 2) ? 1.0 : -1.0;
            int fixed = (f % 2) ? (Nq - 1) : 0;
            for (int t = 0; t < Nq; ++t)
                for (int s = 0; s < Nq; ++s) {
                    int i, j, k;
                    if (a == 0) { i = fixed; j = s; k = t; }
                    else if (a == 1) { i = s; j = fixed; k = t; }
                    else { i = s; j = t; k = fixed; }
                    long p = e * Mn + NODE(i, j, k);
                    if (node) {
                        double gx = met[(3 * a + 0) * NL + p], gy = met[(3 * a + 1) * NL + p],
                               gz = met[(3 * a + 2) * NL + p];
                        double nrm = sqrt(gx * gx + gy * gy + gz * gz);
                        node[cnt] = p;
                        normal[3 * cnt + 0] = sgn * gx / nrm;
                        normal[3 * cnt + 1] = sgn * gy / nrm;
                        normal[3 * cnt + 2] = sgn * gz / nrm;
                    }
                    cnt++;
                }
        }
    return cnt;
}

/* ------------------------------------------------------------------------------------
 * A2-A5  Element-local tendency S(q) of Eq. 1 with H = 0 (DESIGN.md
 * Q18), evaluated as Alg. 1's gradient / divergence / pointwise kernels (L194-L225):
 *
 *   rho = rho0 + rho',  theta = theta0 + theta'
 *   Eq. 3 (L78):  p = p_a (rho R theta / p_a)^gamma,  p' = p - p0,  p0 = EOS(rho0,theta0),
 *       evaluated in the cancellation-free form (Q6)
 *       p' = p0 * expm1( gamma * ( log1p(rho'/rho0) + log1p(theta'/theta0) ) )
 *   gradient (Alg. 2) of the five variables (p', u, v, w, theta)  (L424); theta is
 *       differentiated as theta' plus theta0 separately, grad theta = grad theta' +
 *       grad theta0, both with the same D, theta0 taken relative to its value at the
 *       element's first node (D annihilates the constant; Q7)
 *   chain rule: d f/d x_c = sum_a f_{xi_a} d xi_a/d x_c                  (Q2)
 *   divergence of the momentum F = rho u only (L424): 9 reference derivatives
 *   Eq. 1a:  S_rho   = - div F
 *   Eq. 1b:  S_u     = - u.grad u - grad p'/rho - (rho'/rho) g k,  k = +z  (L66)
 *   Eq. 1c:  S_theta = - u.grad(theta0 + theta')
 *
 * par = {g, p_a, R_gas, c_p, c_v}.  T (optional, may be NULL) receives, per equation and
 * node, the same expression evaluated with every product and every contraction term
 * replaced by its absolute value (sum_l |D f_l| etc.): the quantity that bounds the
 * rounding error of ANY evaluation order, |fl(S) - S| <= c eps T.  It is used only to
 * scale parity errors of fields that are small by cancellation (Q19).
 * ---------------------------------------------------------------------------------- */
void orc_tendency(int N, long Ne, const double *par, const double *q, const double *ref,
                  const double *met, double *S, double *T)
{
    int Nq = N + 1;
    long Mn = (long)Nq * Nq * Nq, NL = Ne * Mn;
    double g = par[0], p_a = par[1], R = par[2], c_p = par[3], c_v = par[4];
    double gamma = c_p / c_v;
    double xi[64], w[64], D[64 * 64];
    orc_lgl(N, xi, w);
    orc_dmat(N, xi, D);
#pragma omp parallel
    {
        /* per-element nodal work arrays: pp, u, v, w, th', th0, Fx, Fy, Fz (+ |p'| scale for T) */
        double *wk = (double *)malloc(sizeof(double) * 10 * Mn);
        double *ppabs = wk + 9 * Mn;
        double *pp = wk, *uu = wk + Mn, *vv = wk + 2 * Mn, *ww = wk + 3 * Mn, *thp = wk + 4 * Mn,
               *th0 = wk + 5 * Mn, *Fx = wk + 6 * Mn, *Fy = wk + 7 * Mn, *Fz = wk + 8 * Mn;
#pragma omp for schedule(static)
        for (long e = 0; e < Ne; ++e) {
            long b = e * Mn;
            for (long n = 0; n < Mn; ++n) {
                double rhop = q[0 * NL + b + n], u = q[1 * NL + b + n], v = q[2 * NL + b + n],
                       wv = q[3 * NL + b + n], tp = q[4 * NL + b + n];
                double rho0 = ref[0 * NL + b + n], theta0 = ref[1 * NL + b + n];
                double rho = rho0 + rhop;
                double p0 = p_a * pow(rho0 * R * theta0 / p_a, gamma);
                pp[n] = p0 * expm1(gamma * (log1p(rhop / rho0) + log1p(tp / theta0)));
                /* scale of p' for T: p' is itself a sum of two terms that may cancel */
                ppabs[n] = p0 * gamma * (fabs(log1p(rhop / rho0)) + fabs(log1p(tp / theta0)));
                uu[n] = u; vv[n] = v; ww[n] = wv; thp[n] = tp; th0[n] = theta0 - ref[1 * NL + b];
                Fx[n] = rho * u; Fy[n] = rho * v; Fz[n] = rho * wv;
            }
            for (int k = 0; k < Nq; ++k)
                for (int j = 0; j < Nq; ++j)
                    for (int i = 0; i < Nq; ++i) {
                        long n = NODE(i, j, k), p = b + n;
                        double m[9];
                        for (int c = 0; c < 9; ++c) m[c] = met[c * NL + p];
                        /* gradients of p', u, v, w, theta', theta0: ref derivs + chain rule */
                        const double *fld[6] = {pp, uu, vv, ww, thp, th0};
                        double grad[6][3];
                        for (int f = 0; f < 6; ++f) {
                            double fx, fe, fz;
                            ref_derivs(Nq, D, fld[f], i, j, k, &fx, &fe, &fz);
                            for (int c = 0; c < 3; ++c)
                                grad[f][c] = fx * m[0 + c] + fe * m[3 + c] + fz * m[6 + c];
                        }
                        /* divergence of F = rho u */
                        const double *F[3] = {Fx, Fy, Fz};
                        double div = 0.0;
                        for (int c = 0; c < 3; ++c) {
                            double fx, fe, fz;
                            ref_derivs(Nq, D, F[c], i, j, k, &fx, &fe, &fz);
                            double d = fx * m[0 + c] + fe * m[3 + c] + fz * m[6 + c];
                            div += d;
                        }
                        double rhop = q[0 * NL + p];
                        double rho = ref[0 * NL + p] + rhop;
                        double u = uu[n], v = vv[n], wv = ww[n];
                        double gth[3] = {grad[4][0] + grad[5][0], grad[4][1] + grad[5][1],
                                         grad[4][2] + grad[5][2]};
                        double advu = u * grad[1][0] + v * grad[1][1] + wv * grad[1][2];
                        double advv = u * grad[2][0] + v * grad[2][1] + wv * grad[2][2];
                        double advw = u * grad[3][0] + v * grad[3][1] + wv * grad[3][2];
                        double advt = u * gth[0] + v * gth[1] + wv * gth[2];
                        S[0 * NL + p] = -div;
                        S[1 * NL + p] = -advu - grad[0][0] / rho;
                        S[2 * NL + p] = -advv - grad[0][1] / rho;
                        S[3 * NL + p] = -advw - grad[0][2] / rho - (rhop / rho) * g;
                        S[4 * NL + p] = -advt;
                        if (T) {
                            double ag[6][3], adv[3] = {fabs(u), fabs(v), fabs(wv)};
                            for (int f = 0; f < 6; ++f) {
                                double ax, ae, az;
                                ref_derivs_abs(Nq, D, f == 0 ? ppabs : fld[f], i, j, k, &ax, &ae, &az);
                                for (int c = 0; c < 3; ++c)
                                    ag[f][c] = ax * fabs(m[0 + c]) + ae * fabs(m[3 + c]) + az * fabs(m[6 + c]);
                            }
                            double adiv2 = 0.0;
                            for (int c = 0; c < 3; ++c) {
                                double ax, ae, az;
                                ref_derivs_abs(Nq, D, F[c], i, j, k, &ax, &ae, &az);
                                adiv2 += ax * fabs(m[0 + c]) + ae * fabs(m[3 + c]) + az * fabs(m[6 + c]);
                            }
                            T[0 * NL + p] = adiv2;
                            for (int c = 0; c < 3; ++c)
                                T[(1 + c) * NL + p] = adv[0] * ag[1 + c][0] + adv[1] * ag[1 + c][1] +
                                                      adv[2] * ag[1 + c][2] + ag[0][c] / rho;
                            T[3 * NL + p] += fabs((rhop / rho) * g);
                            T[4 * NL + p] = adv[0] * (ag[4][0] + ag[5][0]) + adv[1] * (ag[4][1] + ag[5][1]) +
                                            adv[2] * (ag[4][2] + ag[5][2]);
                        }
                    }
        }
        free(wk);
    }
}

/* A6  Local contribution to M^-1 R (Eq. 11-12; Q3):
 * r_loc = (wJ / M_I) * S = omega * S for nf fields. */
void orc_weight(long NL, int nf, const double *omega, const double *S, double *r)
{
    for (int m = 0; m < nf; ++m) {
#pragma omp parallel for schedule(static)
        for (long p = 0; p < NL; ++p) r[m * NL + p] = omega[p] * S[m * NL + p];
    }
}

/* ------------------------------------------------------------------------------------
 * A7  Direct stiffness summation (Eq. 10-11 DSS operator, L115-L121; Alg. 3
 * "Gathering" L263-L270 and "Scattering" L283-L291, single rank so no communication
 * kernel): rhs_cg(I) = sum of rhs over the local copies of I, taken in ascending local
 * index (e, then ijk) order; then every copy receives rhs_cg(I).  In place on r[nf][NL].
 * ---------------------------------------------------------------------------------- */
void orc_dss(long NL, long NG, int nf, const int32_t *intma_cg, double *r)
{
#pragma omp parallel for schedule(static)
    for (int m = 0; m < nf; ++m) {
        double *rhs_cg = (double *)calloc((size_t)NG, sizeof(double));
        double *rm = r + m * NL;
        for (long ip = 0; ip < NL; ++ip) rhs_cg[intma_cg[ip]] = rhs_cg[intma_cg[ip]] + rm[ip];
        for (long ip = 0; ip < NL; ++ip) rm[ip] = rhs_cg[intma_cg[ip]];
        free(rhs_cg);
    }
}

/* ------------------------------------------------------------------------------------
 * A8  Pointwise sources added to the assembled tendency (Q9, Q10, Q15):
 *   heating S_theta of Eq. 1c:           r_theta += heat
 *   f-plane Coriolis (config 3; absent from Eq. 1b):          r_u += f v,  r_v -= f u
 *   Rayleigh sponge (explicit stand-in for L256's layer):     r_m -= beta q_m, m = u,v,w,theta'
 * heat and beta may be NULL.
 * ---------------------------------------------------------------------------------- */
void orc_sources(long NL, const double *q, const double *heat, const double *beta, double f_cor,
                 double *r)
{
#pragma omp parallel for schedule(static)
    for (long p = 0; p < NL; ++p) {
        double u = q[1 * NL + p], v = q[2 * NL + p];
        if (heat) r[4 * NL + p] += heat[p];
        r[1 * NL + p] += f_cor * v;
        r[2 * NL + p] -= f_cor * u;
        if (beta) {
            double b = beta[p];
            r[1 * NL + p] -= b * u;
            r[2 * NL + p] -= b * v;
            r[3 * NL + p] -= b * q[3 * NL + p];
            r[4 * NL + p] -= b * q[4 * NL + p];
        }
    }
}

/* A9  No-flux walls (Q8): for each wall entry, in list order,
 * remove the normal component of the velocity tendency: r_vel -= (r_vel . n) n. */
void orc_walls(long NL, long n_wall, const int64_t *node, const double *normal, double *r)
{
    for (long t = 0; t < n_wall; ++t) {
        long p = node[t];
        const double *n = normal + 3 * t;
        double rn = r[1 * NL + p] * n[0] + r[2 * NL + p] * n[1] + r[3 * NL + p] * n[2];
        r[1 * NL + p] -= rn * n[0];
        r[2 * NL + p] -= rn * n[1];
        r[3 * NL + p] -= rn * n[2];
    }
}

/* A10  Explicit Runge-Kutta stage update ("updating the state vector", PAPER.md:L172;
 * scheme per DESIGN.md Q11): q_out = a0 q0 + a1 qs + b_dt r, for n values.
 * q_out may alias q0 or qs. */
void orc_rk_stage(long n, double a0, double a1, double b_dt, const double *q0, const double *qs,
                  const double *r, double *q_out)
{
#pragma omp parallel for schedule(static)
    for (long p = 0; p < n; ++p) q_out[p] = a0 * q0[p] + a1 * qs[p] + b_dt * r[p];
}

/* ------------------------------------------------------------------------------------
 * NEXT-4  RI-velocity diagnostic (Eq. 18-22; readings Q25-Q29 of
 * DESIGN.md).  Pins: tests/test_oracle_ri.py.
 *
 * orc_ri_area: horizontal quadrature weight of every local node,
 *     a = w_i w_j |x_xi y_eta - x_eta y_xi|,
 * the LGL quadrature (Eq. 8) of the level surface zeta = const of a
 * column-preserving mesh (L162-L168); the integrals "int_x int_y ... dx dy" of Eq. 22 at
 * a height z are sums over the local nodes of that level with this weight (Q26).
 * ---------------------------------------------------------------------------------- */
void orc_ri_area(int N, long Ne, const double *xyz, double *a)
{
    int Nq = N + 1;
    long Mn = (long)Nq * Nq * Nq, NL = Ne * Mn;
    double xi[64], w[64], D[64 * 64];
    orc_lgl(N, xi, w);
    orc_dmat(N, xi, D);
    for (long e = 0; e < Ne; ++e) {
        const double *x = xyz + 0 * NL + e * Mn, *y = xyz + 1 * NL + e * Mn;
        for (int k = 0; k < Nq; ++k)
            for (int j = 0; j < Nq; ++j)
                for (int i = 0; i < Nq; ++i) {
                    double xx, xe, xz, yx, ye, yz;
                    ref_derivs_diff(Nq, D, x, i, j, k, &xx, &xe, &xz);
                    ref_derivs_diff(Nq, D, y, i, j, k, &yx, &ye, &yz);
                    a[e * Mn + NODE(i, j, k)] = w[i] * w[j] * fabs(xx * ye - xe * yx);
                }
    }
}

/* orc_ri_velocity, in the paper's order:
 *  Eq. 22 (L352): per level l, x_c = sum a |u| x / sum a |u|, |u| = (u^2+v^2+w^2)^(1/2)
 *      ("weighted center of the velocity magnitude field", vertically varying); a level
 *      whose denominator is 0 has no centroid and takes no part (valid[l] = 0).
 *  Eq. 21 (L346): u_theta = (I - e_r x e_r - e_z x e_z) u,  e_r = r/|r|,
 *      r = (x - x_c, y - y_c, 0), e_z = (0,0,1);   Eq. 20: u_theta = |u_theta| (a norm).
 *  Strip mean (L360-L364): arithmetic mean of u_theta over the POINTS of the strip
 *      s eps <= r < (s+1) eps, eps = r_max / n_strip, at each level (50 equi-width strips,
 *      L366).  A point = a unique global node (its first local copy, Q28); a point with
 *      r = 0 has no radial direction, nothing radial is removed there (e_r := 0) and it
 *      belongs to strip 0; points with r >= r_max are left out (Q29).
 *  Eq. 18 (L338): u_RI = max over (strip, level) with at least one point.
 *  scalars[0] = u_RI, scalars[1] = max over points of (u^2+v^2)^(1/2) ("maximum horizontal
 *      velocity" of Fig. 9).
 * ---------------------------------------------------------------------------------- */
void orc_ri_velocity(long NL, long NG, const int32_t *intma_cg, const int32_t *level, int n_lev,
                     int n_strip, double r_max, const double *xyz, const double *a,
                     const double *q, double *centroid /* [n_lev][2] */, int32_t *valid /* [n_lev] */,
                     double *ubar /* [n_lev][n_strip] */, int32_t *count /* [n_lev][n_strip] */,
                     double *scalars /* [2] */)
{
    const double *x = xyz, *y = xyz + NL;
    const double *u = q + 1 * NL, *v = q + 2 * NL, *w = q + 3 * NL;
    double *num_x = (double *)calloc((size_t)n_lev, sizeof(double));
    double *num_y = (double *)calloc((size_t)n_lev, sizeof(double));
    double *den = (double *)calloc((size_t)n_lev, sizeof(double));
    for (long p = 0; p < NL; ++p) {
        int l = level[p];
        double mag = sqrt(u[p] * u[p] + v[p] * v[p] + w[p] * w[p]);
        num_x[l] += a[p] * mag * x[p];
        num_y[l] += a[p] * mag * y[p];
        den[l] += a[p] * mag;
    }
    for (int l = 0; l < n_lev; ++l) {
        valid[l] = den[l] > 0.0;
        centroid[2 * l + 0] = valid[l] ? num_x[l] / den[l] : 0.0;
        centroid[2 * l + 1] = valid[l] ? num_y[l] / den[l] : 0.0;
    }
    for (long t = 0; t < (long)n_lev * n_strip; ++t) { ubar[t] = 0.0; count[t] = 0; }
    char *seen = (char *)calloc((size_t)NG, 1);
    double eps = r_max / n_strip, umax_h = 0.0;
    for (long p = 0; p < NL; ++p) {
        long I = intma_cg[p];
        if (seen[I]) continue;   /* a point is a unique global node: its first local copy */
        seen[I] = 1;
        double uh = sqrt(u[p] * u[p] + v[p] * v[p]);
        if (uh > umax_h) umax_h = uh;
        int l = level[p];
        if (!valid[l]) continue;
        double rx = x[p] - centroid[2 * l + 0], ry = y[p] - centroid[2 * l + 1];
        double r = sqrt(rx * rx + ry * ry);
        if (!(r < r_max)) continue;
        double er[3] = {0.0, 0.0, 0.0}, ez[3] = {0.0, 0.0, 1.0};
        if (r > 0.0) { er[0] = rx / r; er[1] = ry / r; }
        double uu[3] = {u[p], v[p], w[p]};
        double ur = uu[0] * er[0] + uu[1] * er[1] + uu[2] * er[2];
        double uz = uu[0] * ez[0] + uu[1] * ez[1] + uu[2] * ez[2];
        double t0 = uu[0] - ur * er[0] - uz * ez[0];
        double t1 = uu[1] - ur * er[1] - uz * ez[1];
        double t2 = uu[2] - ur * er[2] - uz * ez[2];
        double ut = sqrt(t0 * t0 + t1 * t1 + t2 * t2);
        int s = (int)floor(r / eps);
        if (s >= n_strip) continue;
        ubar[(long)l * n_strip + s] += ut;
        count[(long)l * n_strip + s] += 1;
    }
    double uri = 0.0;
    for (long t = 0; t < (long)n_lev * n_strip; ++t)
        if (count[t] > 0) {
            ubar[t] /= count[t];
            if (ubar[t] > uri) uri = ubar[t];
        }
    scalars[0] = uri;
    scalars[1] = umax_h;
    free(seen); free(num_x); free(num_y); free(den);
}

/* ------------------------------------------------------------------------------------
 * NEXT-1  Tensor-based hyper-diffusion (Section 2.4, Eq. 14-16;
 * readings Q30-Q33 of DESIGN.md).  H_q = (-1)^(alpha+1) (div tau grad)^alpha q with
 * alpha = 2 (L145): H_q = - L(L(q)),  L f = div( tau grad f ), tau applied in EACH
 * application of the Laplacian (L145 "multiplying the viscosity tensor tau by each
 * application of the Laplacian operator").  The viscosity tensor tau (Eq. 15-16) is built in
 * oracle.py with LAPACK's symmetric eigensolver as the library step.
 *
 * orc_hd_laplacian: element-local strong form, in the same style as Alg. 1-2 (Q2, Q30):
 *   g   = grad f           (Alg. 2 reference derivatives + chain rule with grad xi_a)
 *   F   = tau g            (tau[6][NL] = xx, xy, xz, yy, yz, zz at every local node)
 *   out = div F            (9 reference derivatives + chain rule), for nf fields.
 * The assembly between and after the two applications (omega weight + DSS, Eq. 11-12) is
 * done by the caller with orc_weight / orc_dss.  Pins: tests/test_oracle_hyperdiffusion.py.
 * ---------------------------------------------------------------------------------- */
void orc_hd_laplacian(int N, long Ne, int nf, const double *met, const double *tau, const double *f,
                      double *out)
{
    int Nq = N + 1;
    long Mn = (long)Nq * Nq * Nq, NL = Ne * Mn;
    double xi[64], w[64], D[64 * 64];
    orc_lgl(N, xi, w);
    orc_dmat(N, xi, D);
#pragma omp parallel
    {
        double *F = (double *)malloc(sizeof(double) * 3 * Mn);
#pragma omp for schedule(static)
        for (long e = 0; e < Ne; ++e) {
            long b = e * Mn;
            for (int m = 0; m < nf; ++m) {
                const double *fe = f + (long)m * NL + b;
                for (int k = 0; k < Nq; ++k)
                    for (int j = 0; j < Nq; ++j)
                        for (int i = 0; i < Nq; ++i) {
                            long n = NODE(i, j, k), p = b + n;
                            double fx, fy, fz, g[3];
                            ref_derivs(Nq, D, fe, i, j, k, &fx, &fy, &fz);
                            for (int c = 0; c < 3; ++c)
                                g[c] = fx * met[(0 + c) * NL + p] + fy * met[(3 + c) * NL + p] +
                                       fz * met[(6 + c) * NL + p];
                            double txx = tau[0 * NL + p], txy = tau[1 * NL + p], txz = tau[2 * NL + p],
                                   tyy = tau[3 * NL + p], tyz = tau[4 * NL + p], tzz = tau[5 * NL + p];
                            F[0 * Mn + n] = txx * g[0] + txy * g[1] + txz * g[2];
                            F[1 * Mn + n] = txy * g[0] + tyy * g[1] + tyz * g[2];
                            F[2 * Mn + n] = txz * g[0] + tyz * g[1] + tzz * g[2];
                        }
                for (int k = 0; k < Nq; ++k)
                    for (int j = 0; j < Nq; ++j)
                        for (int i = 0; i < Nq; ++i) {
                            long p = b + NODE(i, j, k);
                            double div = 0.0;
                            for (int c = 0; c < 3; ++c) {
                                double fx, fy, fz;
                                ref_derivs(Nq, D, F + c * Mn, i, j, k, &fx, &fy, &fz);
                                div += fx * met[(0 + c) * NL + p] + fy * met[(3 + c) * NL + p] +
                                       fz * met[(6 + c) * NL + p];
                            }
                            out[(long)m * NL + p] = div;
                        }
            }
        }
        free(F);
    }
}

/* ------------------------------------------------------------------------------------
 * NEXT-3  Linear operator of the IMEX splitting (Section 2.3, Eq. 13):
 *     dq/dt = [S(q) - L(q)] + L(q),
 * "the linear operator L(q) represent[s] fast waves, such as acoustic and gravity waves".
 * The paper does not print L (it cites Giraldo et al. 2013); reading Q34 of DESIGN.md: L is the
 * linearisation (Jacobian) of the S of Eq. 1 about the hydrostatic reference state q = 0,
 *     L_rho   = - div( rho0 u )
 *     L_u     = - grad p'_L / rho0 - (rho'/rho0) g k,
 *               p'_L = gamma p0 ( rho'/rho0 + theta'/theta0 )   (Eq. 3 linearised; p0 = EOS(rho0,theta0))
 *     L_theta = - u . grad theta0
 * evaluated element-locally exactly as orc_tendency evaluates S (Alg. 2 derivatives + chain
 * rule, Q2; grad theta0 relative to the element's first node, Q7).  Pinned as the directional
 * derivative of orc_tendency: L(v) = lim S(eps v)/eps (tests/test_oracle_imex.py).
 * ---------------------------------------------------------------------------------- */
void orc_linear_tendency(int N, long Ne, const double *par, const double *q, const double *ref,
                         const double *met, double *Lq)
{
    int Nq = N + 1;
    long Mn = (long)Nq * Nq * Nq, NL = Ne * Mn;
    double g = par[0], p_a = par[1], R = par[2], c_p = par[3], c_v = par[4];
    double gamma = c_p / c_v;
    double xi[64], w[64], D[64 * 64];
    orc_lgl(N, xi, w);
    orc_dmat(N, xi, D);
#pragma omp parallel
    {
        double *wk = (double *)malloc(sizeof(double) * 5 * Mn);
        double *pl = wk, *th0 = wk + Mn, *Fx = wk + 2 * Mn, *Fy = wk + 3 * Mn, *Fz = wk + 4 * Mn;
#pragma omp for schedule(static)
        for (long e = 0; e < Ne; ++e) {
            long b = e * Mn;
            for (long n = 0; n < Mn; ++n) {
                double rho0 = ref[0 * NL + b + n], theta0 = ref[1 * NL + b + n];
                double p0 = p_a * pow(rho0 * R * theta0 / p_a, gamma);
                pl[n] = gamma * p0 * (q[0 * NL + b + n] / rho0 + q[4 * NL + b + n] / theta0);
                th0[n] = theta0 - ref[1 * NL + b];
                Fx[n] = rho0 * q[1 * NL + b + n];
                Fy[n] = rho0 * q[2 * NL + b + n];
                Fz[n] = rho0 * q[3 * NL + b + n];
            }
            for (int k = 0; k < Nq; ++k)
                for (int j = 0; j < Nq; ++j)
                    for (int i = 0; i < Nq; ++i) {
                        long p = b + NODE(i, j, k);
                        double m[9];
                        for (int c = 0; c < 9; ++c) m[c] = met[c * NL + p];
                        double fx, fe, fz, gp[3], gt[3], div = 0.0;
                        ref_derivs(Nq, D, pl, i, j, k, &fx, &fe, &fz);
                        for (int c = 0; c < 3; ++c) gp[c] = fx * m[0 + c] + fe * m[3 + c] + fz * m[6 + c];
                        ref_derivs(Nq, D, th0, i, j, k, &fx, &fe, &fz);
                        for (int c = 0; c < 3; ++c) gt[c] = fx * m[0 + c] + fe * m[3 + c] + fz * m[6 + c];
                        const double *F[3] = {Fx, Fy, Fz};
                        for (int c = 0; c < 3; ++c) {
                            ref_derivs(Nq, D, F[c], i, j, k, &fx, &fe, &fz);
                            div += fx * m[0 + c] + fe * m[3 + c] + fz * m[6 + c];
                        }
                        double rho0 = ref[0 * NL + p];
                        double u = q[1 * NL + p], v = q[2 * NL + p], wv = q[3 * NL + p];
                        Lq[0 * NL + p] = -div;
                        Lq[1 * NL + p] = -gp[0] / rho0;
                        Lq[2 * NL + p] = -gp[1] / rho0;
                        Lq[3 * NL + p] = -gp[2] / rho0 - (q[0 * NL + p] / rho0) * g;
                        Lq[4 * NL + p] = -(u * gt[0] + v * gt[1] + wv * gt[2]);
                    }
        }
        free(wk);
    }
}
