/*
 * lbwp_oracle.c -- CPU ORACLE for "LB without populations" (arxiv 2301.01622).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, fp64,
 * loop-nest restatement of the paper's equations, written to be checked
 * against PAPER.md by eye.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load it.  It shares no
 * code, header, table or constant generator with the CUDA path under
 * paper_2301_01622_b200/csrc/.
 *
 * Citations are "PAPER.md:<line>" (+ equation); readings Cn are the ones
 * listed in DESIGN.md "Readings of the paper".
 *
 * Parity pins (tests/test_oracle_*.py):
 *   single-component step .......... pinned (round trip, fixed point,
 *       conservation, Taylor-Green viscosity, tau=1, lattice symmetry,
 *       independent numpy regularised-BGK-with-populations, dense brute force)
 *   two-component colour-gradient .. the operator formulas are not printed in
 *       the paper (PAPER.md:91 defers to ref. [25]); reading C6 is pinned by
 *       what the mathematics fixes: A=0 reduction, colour mass and momentum
 *       conservation, uniform mixture, Laplace law sigma = (2/9) A tau, and the
 *       exact steady flat-interface balance phi(x+1)-phi(x) = (3 beta kappa_L/2)
 *       [(1-phi(x)^2)+(1-phi(x+1)^2)], kappa_L = sum_i w_i c_ix^2/|c_i| (fixes
 *       beta, the 1/|c_i| of cos(theta_i), the w_i rho factor and the sign of
 *       the recolouring term); the |G|->0 constant of C8 is bracketed (sigma
 *       independent of it, spurious currents not).  Against the paper's own
 *       code and figures: PARITY UNPINNED.
 *   population-storing BGK (comparison kernel's mini-oracle): conservation +
 *       Taylor-Green viscosity (ncomp=1); ncomp=2: equality with the moments
 *       run at tau=1, per-colour mass conservation, A=0 reduction to ncomp=1.
 *
 * Layout of every moment array: dense SoA [M][nz][ny][nx], x fastest.
 *   M = 10 : rho, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz          (C11, C12)
 *   M = 11 : rhoA, rhoB, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz
 * P is the full second moment sum_i f_i c_ia c_ib (Eq. 3).
 *
 * Thread count: the loop over z carries an OpenMP pragma; each node's result
 * is computed by one thread from read-only input, so the output is
 * bit-identical for any number of threads.  Compiled without -fopenmp it is
 * the single-threaded program the north star describes.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define CS2 (1.0 / 3.0) /* cs^2 = 1/3 */

/* ------------------------------------------------------------------------ */
/* Lattice tables (textbook; "w_i ... depend on the lattice      */
/* geometry").  Direction order: lexicographic in (cz, cy, cx), -1..1.       */
/* D3Q27: all 27 vectors, w = 8/27, 2/27, 1/54, 1/216 by |c|^2 = 0,1,2,3.    */
/* D3Q19: |c|^2 <= 2,     w = 1/3, 1/18, 1/36.                               */
/* ------------------------------------------------------------------------ */
typedef struct {
    int q;
    int c[27][3];
    double w[27];
} lattice_t;

static int lattice_make(int lattice, lattice_t *L) {
    if (lattice != 19 && lattice != 27) return -1;
    int n = 0;
    for (int cz = -1; cz <= 1; ++cz)
        for (int cy = -1; cy <= 1; ++cy)
            for (int cx = -1; cx <= 1; ++cx) {
                int n2 = cx * cx + cy * cy + cz * cz;
                if (lattice == 19 && n2 == 3) continue;
                L->c[n][0] = cx;
                L->c[n][1] = cy;
                L->c[n][2] = cz;
                if (lattice == 27) {
                    const double wt[4] = {8.0 / 27.0, 2.0 / 27.0, 1.0 / 54.0, 1.0 / 216.0};
                    L->w[n] = wt[n2];
                } else {
                    const double wt[3] = {1.0 / 3.0, 1.0 / 18.0, 1.0 / 36.0};
                    L->w[n] = wt[n2];
                }
                ++n;
            }
    L->q = n;
    return 0;
}

int lbwp_oracle_lattice(int lattice, int *c_out /* [Q][3] */, double *w_out /* [Q] */) {
    lattice_t L;
    if (lattice_make(lattice, &L)) return -1;
    for (int i = 0; i < L.q; ++i) {
        for (int a = 0; a < 3; ++a) c_out[3 * i + a] = L.c[i][a];
        w_out[i] = L.w[i];
    }
    return L.q;
}

/* index of the symmetric pair (a,b) in the stored order xx,yy,zz,xy,xz,yz (C12) */
static const int PIDX[3][3] = {{0, 3, 4}, {3, 1, 5}, {4, 5, 2}};

/* Q_iab = (c_ia c_ib - cs^2 delta_ab) / (2 cs^4)   (reading C1) */
static double Qiab(const int *c, int a, int b) {
    return ((double)(c[a] * c[b]) - (a == b ? CS2 : 0.0)) / (2.0 * CS2 * CS2);
}

/* ------------------------------------------------------------------------ */
/* Eq. 8, one direction:                                    */
/*   h'_i = w_i rho (1 + c_i.u/cs^2 + Q_iab u_a u_b)                          */
/*        + (1-omega) w_i Q_iab (P_ab - P^eq_ab)                              */
/* with P^eq_ab = rho cs^2 delta_ab + rho u_a u_b (reading C2).              */
/* omega = 0 gives Eq. 4 (the reconstruction h_i itself).                    */
/* The double contraction runs over the full 3x3 (off-diagonals twice).      */
/* ------------------------------------------------------------------------ */
static double hprime(const lattice_t *L, int i, double rho, const double u[3], const double P[6],
                     double omega) {
    const int *c = L->c[i];
    double cu = 0.0;
    for (int a = 0; a < 3; ++a) cu += c[a] * u[a];
    double quu = 0.0, qneq = 0.0;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            double q = Qiab(c, a, b);
            double peq = rho * u[a] * u[b] + (a == b ? rho * CS2 : 0.0);
            quu += q * u[a] * u[b];
            qneq += q * (P[PIDX[a][b]] - peq);
        }
    double heq = L->w[i] * rho * (1.0 + cu / CS2 + quu);  /* Eq. 5 */
    double hneq = L->w[i] * qneq;                          /* Eq. 6 */
    return heq + (1.0 - omega) * hneq;                     /* Eq. 8 */
}

/* h_i for all directions from one node's moments H = (rho,u,P); omega as above. */
int lbwp_oracle_reconstruct(int lattice, const double *H10, double omega, double *h_out) {
    lattice_t L;
    if (lattice_make(lattice, &L)) return -1;
    for (int i = 0; i < L.q; ++i) h_out[i] = hprime(&L, i, H10[0], H10 + 1, H10 + 4, omega);
    return L.q;
}

/* Eq. 1-3: H = P f for one node; returns rho, u (=j/rho), P. */
int lbwp_oracle_project(int lattice, const double *f, double *H10) {
    lattice_t L;
    if (lattice_make(lattice, &L)) return -1;
    double rho = 0.0, j[3] = {0, 0, 0}, P[6] = {0, 0, 0, 0, 0, 0};
    for (int i = 0; i < L.q; ++i) {
        const int *c = L.c[i];
        rho += f[i];
        for (int a = 0; a < 3; ++a) j[a] += f[i] * c[a];
        for (int a = 0; a < 3; ++a)
            for (int b = a; b < 3; ++b) P[PIDX[a][b]] += f[i] * c[a] * c[b];
    }
    H10[0] = rho;
    for (int a = 0; a < 3; ++a) H10[1 + a] = j[a] / rho;
    for (int k = 0; k < 6; ++k) H10[4 + k] = P[k];
    return 0;
}

static inline int wrap(int i, int n) { /* periodic box, reading C13 */
    i %= n;
    return i < 0 ? i + n : i;
}

/* ------------------------------------------------------------------------ */
/* Single-component fused step (Eq. 8, 9, 1-3).          */
/* For every node x: for every direction i, y = x - c_i (periodic);          */
/* h'_i from the moments stored at y (Eq. 8); it arrives at x (Eq. 9);       */
/* new moments at x are the sums Eq. 1-3 of the arrived populations.         */
/* Stored moments are post-stream, pre-collision (reading C5).               */
/* ------------------------------------------------------------------------ */
static void step_1c(const lattice_t *L, int nx, int ny, int nz, double omega, const double *src,
                    double *dst) {
    const size_t n = (size_t)nx * ny * nz;
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double rho = 0.0, j[3] = {0, 0, 0}, P[6] = {0, 0, 0, 0, 0, 0};
                for (int i = 0; i < L->q; ++i) {
                    const int *c = L->c[i];
                    size_t yy = ((size_t)wrap(z - c[2], nz) * ny + wrap(y - c[1], ny)) * nx +
                                wrap(x - c[0], nx);
                    double u[3], Pn[6];
                    for (int a = 0; a < 3; ++a) u[a] = src[(1 + a) * n + yy];
                    for (int k = 0; k < 6; ++k) Pn[k] = src[(4 + k) * n + yy];
                    double h = hprime(L, i, src[yy], u, Pn, omega);
                    rho += h;                                       /* Eq. 1 */
                    for (int a = 0; a < 3; ++a) j[a] += h * c[a];   /* Eq. 2 */
                    for (int a = 0; a < 3; ++a)                     /* Eq. 3 */
                        for (int b = a; b < 3; ++b) P[PIDX[a][b]] += h * c[a] * c[b];
                }
                size_t xx = ((size_t)z * ny + y) * nx + x;
                dst[xx] = rho;
                for (int a = 0; a < 3; ++a) dst[(1 + a) * n + xx] = j[a] / rho; /* C11 */
                for (int k = 0; k < 6; ++k) dst[(4 + k) * n + xx] = P[k];
            }
}

/* ------------------------------------------------------------------------ */
/* Two-component colour-gradient step (reading C6/C7/C8,    */
/* 105).  State: rhoA, rhoB, u, P (u, P of the total fluid).                 */
/*  0. phi = (rhoA-rhoB)/(rhoA+rhoB);                         */
/*     G(y) = (1/cs^2) sum_i w_i c_i phi(y+c_i); n = G/|G| (0 if |G|^2<=1e-10)*/
/*  1. at y = x-c_i: h' by Eq. 8 with rho = rhoA+rhoB;                       */
/*     perturbation  h'' = h' + (A/2)|G| [ w_i (c_i.n)^2 - B_i ],            */
/*        B_i = w_i (i != rest), B_0 = w_0 - 2/3;                            */
/*     recolouring   hA = (rhoA/rho) h'' + beta (rhoA rhoB/rho^2) cos_i w_i rho,*/
/*        cos_i = (c_i.n)/|c_i| (0 for rest);  hB = h'' - hA;                */
/*     accumulate rhoA += hA, rhoB += hB, j += h'' c_i, P += h'' c_i c_i.    */
/*  2. u = j/(rhoA+rhoB).                                                    */
/* Order BGK -> perturbation -> recolouring is PAPER.md:91.                  */
/* grad is scratch of 4*n doubles: Gx, Gy, Gz, (unused).                     */
/* ------------------------------------------------------------------------ */
static void colour_gradient(const lattice_t *L, int nx, int ny, int nz, const double *rhoA,
                            const double *rhoB, double *grad) {
    const size_t n = (size_t)nx * ny * nz;
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double G[3] = {0, 0, 0};
                for (int i = 0; i < L->q; ++i) {
                    const int *c = L->c[i];
                    size_t yy = ((size_t)wrap(z + c[2], nz) * ny + wrap(y + c[1], ny)) * nx +
                                wrap(x + c[0], nx);
                    double phi = (rhoA[yy] - rhoB[yy]) / (rhoA[yy] + rhoB[yy]);
                    for (int a = 0; a < 3; ++a) G[a] += L->w[i] * c[a] * phi;
                }
                size_t xx = ((size_t)z * ny + y) * nx + x;
                for (int a = 0; a < 3; ++a) grad[a * n + xx] = G[a] / CS2;
            }
}

/* Reading C8: n = G/|G| where |G|^2 > g2cut, else n = 0 (the paper is silent on |G| -> 0).
 * 1e-10 is the value every parity run uses; it was taken after the fp32 kernel existed (|G| <= 1e-5
 * is below the fp32 rounding noise of phi), SURVEY proposed 1e-30.  lbwp_oracle_set_g2cut() exists
 * only so that a pin can bracket what depends on the choice (tests/test_oracle_pins_two_component.py:
 * the Laplace-law sigma does not, the spurious currents do). */
static double g2cut = 1e-10;
void lbwp_oracle_set_g2cut(double v) { g2cut = v; }
double lbwp_oracle_get_g2cut(void) { return g2cut; }

/* perturbation + recolouring of one population (shared by the moments oracle
 * and the population-storing comparison oracle: same reading C6). */
static void colour_ops(const lattice_t *L, int i, double hp, double rhoA, double rhoB,
                       const double G[3], double A, double beta, double *hA, double *hB) {
    const int *c = L->c[i];
    double g2 = G[0] * G[0] + G[1] * G[1] + G[2] * G[2];
    double gn = 0.0, nvec[3] = {0, 0, 0};
    if (g2 > g2cut) { /* C8 (default 1e-10: |G| <= 1e-5 is below the fp32 noise of phi); n := 0 */
        gn = sqrt(g2);
        for (int a = 0; a < 3; ++a) nvec[a] = G[a] / gn;
    }
    double cn = c[0] * nvec[0] + c[1] * nvec[1] + c[2] * nvec[2];
    int c2 = c[0] * c[0] + c[1] * c[1] + c[2] * c[2];
    double Bi = (c2 == 0) ? L->w[i] - 2.0 / 3.0 : L->w[i];
    double hpp = hp + 0.5 * A * gn * (L->w[i] * cn * cn - Bi);
    double rho = rhoA + rhoB;
    double cosi = (c2 == 0) ? 0.0 : cn / sqrt((double)c2);
    *hA = (rhoA / rho) * hpp + beta * (rhoA * rhoB / (rho * rho)) * cosi * L->w[i] * rho;
    *hB = hpp - *hA;
}

static void step_2c(const lattice_t *L, int nx, int ny, int nz, double omega, double A,
                    double beta, const double *src, double *dst, double *grad) {
    const size_t n = (size_t)nx * ny * nz;
    colour_gradient(L, nx, ny, nz, src, src + n, grad);
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double rA = 0.0, rB = 0.0, j[3] = {0, 0, 0}, P[6] = {0, 0, 0, 0, 0, 0};
                for (int i = 0; i < L->q; ++i) {
                    const int *c = L->c[i];
                    size_t yy = ((size_t)wrap(z - c[2], nz) * ny + wrap(y - c[1], ny)) * nx +
                                wrap(x - c[0], nx);
                    double u[3], Pn[6], G[3];
                    double a_ = src[yy], b_ = src[n + yy];
                    for (int a = 0; a < 3; ++a) u[a] = src[(2 + a) * n + yy];
                    for (int k = 0; k < 6; ++k) Pn[k] = src[(5 + k) * n + yy];
                    for (int a = 0; a < 3; ++a) G[a] = grad[a * n + yy];
                    double hp = hprime(L, i, a_ + b_, u, Pn, omega);
                    double hA, hB;
                    colour_ops(L, i, hp, a_, b_, G, A, beta, &hA, &hB);
                    double hpp = hA + hB;
                    rA += hA;
                    rB += hB;
                    for (int a = 0; a < 3; ++a) j[a] += hpp * c[a];
                    for (int a = 0; a < 3; ++a)
                        for (int b = a; b < 3; ++b) P[PIDX[a][b]] += hpp * c[a] * c[b];
                }
                size_t xx = ((size_t)z * ny + y) * nx + x;
                dst[xx] = rA;
                dst[n + xx] = rB;
                for (int a = 0; a < 3; ++a) dst[(2 + a) * n + xx] = j[a] / (rA + rB);
                for (int k = 0; k < 6; ++k) dst[(5 + k) * n + xx] = P[k];
            }
}

/* ------------------------------------------------------------------------ */
/* Near-contact repulsion (Eq. 10):                          */
/*     F_rep = - A_h[h(x)] n delta_I .                                        */
/* The paper gives neither h(x) nor the forcing scheme (both are in its ref.  */
/* [26]); readings C20-C24 of DESIGN.md, PARITY WITH THE PAPER'S CODE         */
/* UNPINNED:                                                                  */
/*  C20 delta_I = |grad phi| / 2 = |G|/2 (integrates to 1 across an interface)*/
/*  C21 n = outward unit normal of the droplet phase = -G/|G| (phi = +1       */
/*      inside), so F_rep = (A_h/2) G: it pushes an interface away from the   */
/*      one it faces.                                                         */
/*  C22 h(x), at INTERFACE nodes, |G| > G_I = 0.05 (a tenth of the peak        */
/*      gradient 1/W of a tanh interface of width W = 2): walk from x along    */
/*      the lattice direction c_m closest to n (largest c.n/|c|; first in      */
/*      direction order on a tie), p_k = x + k c_m, k = 1, 2, ... while        */
/*      k |c_m| <= h_c; the first interface node p_k whose gradient opposes    */
/*      G (G(p_k).G(x) < 0, |G(p_k)| > G_I) is a facing interface and          */
/*      h = k |c_m|; none: h = infinity.                                       */
/*  C23 A_h[h] = A_h for h <= h_c, 0 beyond (one strength).     */
/*  C24 forcing in moment space: Guo's scheme on the reconstructed            */
/*      populations, see hprime_forced().                                     */
/* force: 3*n doubles Fx, Fy, Fz.                                             */
/* ------------------------------------------------------------------------ */
#define G_I2 (0.05 * 0.05)
static void contact_force(const lattice_t *L, int nx, int ny, int nz, const double *grad, double A_h,
                          double h_c, double *force) {
    const size_t n = (size_t)nx * ny * nz;
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const size_t xx = ((size_t)z * ny + y) * nx + x;
                double G[3] = {grad[xx], grad[n + xx], grad[2 * n + xx]};
                double F[3] = {0, 0, 0};
                const double g2 = G[0] * G[0] + G[1] * G[1] + G[2] * G[2];
                if (g2 > G_I2 && A_h != 0.0) {
                    int m = -1;
                    double best = -1e300;
                    for (int i = 0; i < L->q; ++i) { /* lattice direction closest to n = -G/|G| */
                        const int *c = L->c[i];
                        const int c2 = c[0] * c[0] + c[1] * c[1] + c[2] * c[2];
                        if (c2 == 0) continue;
                        const double cosv = -(c[0] * G[0] + c[1] * G[1] + c[2] * G[2]) / sqrt((double)c2);
                        if (cosv > best) { best = cosv; m = i; }
                    }
                    const int *c = L->c[m];
                    const double len = sqrt((double)(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]));
                    for (int k = 1; k * len <= h_c; ++k) {
                        const size_t pp = ((size_t)wrap(z + k * c[2], nz) * ny + wrap(y + k * c[1], ny)) * nx +
                                          wrap(x + k * c[0], nx);
                        const double Gp[3] = {grad[pp], grad[n + pp], grad[2 * n + pp]};
                        const double gp2 = Gp[0] * Gp[0] + Gp[1] * Gp[1] + Gp[2] * Gp[2];
                        if (gp2 > G_I2 && Gp[0] * G[0] + Gp[1] * G[1] + Gp[2] * G[2] < 0.0) {
                            for (int a = 0; a < 3; ++a) F[a] = 0.5 * A_h * G[a]; /* -A_h n delta_I */
                            break;
                        }
                    }
                }
                for (int a = 0; a < 3; ++a) force[a * n + xx] = F[a];
            }
}

/* Eq. 8 with a body force F (reading C24): Guo, Zheng and Shi's forcing on the   */
/* reconstructed populations.  u* = u + F/(2 rho) is the velocity of the         */
/* equilibrium; the stored first moment rho u differs from rho u* by -F/2, a     */
/* first-order non-equilibrium part that relaxes like the second-order one;      */
/* S_i = (1 - omega/2) w_i [ (c_i - u*)/cs^2 + (c_i.u*) c_i / cs^4 ] . F.         */
/* Its moments: sum_i = rho, sum_i c_i = rho u + F (momentum gains F per step),  */
/* F = 0 gives hprime().                                                         */
static double hprime_forced(const lattice_t *L, int i, double rho, const double u[3], const double P[6],
                            double omega, const double F[3]) {
    const int *c = L->c[i];
    double us[3], cu = 0.0, cF = 0.0, uF = 0.0, cdu = 0.0;
    for (int a = 0; a < 3; ++a) us[a] = u[a] + F[a] / (2.0 * rho);
    for (int a = 0; a < 3; ++a) {
        cu += c[a] * us[a];
        cF += c[a] * F[a];
        uF += us[a] * F[a];
        cdu += c[a] * (rho * u[a] - rho * us[a]);
    }
    double quu = 0.0, qneq = 0.0;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            double q = Qiab(c, a, b);
            double peq = rho * us[a] * us[b] + (a == b ? rho * CS2 : 0.0);
            quu += q * us[a] * us[b];
            qneq += q * (P[PIDX[a][b]] - peq);
        }
    double heq = L->w[i] * rho * (1.0 + cu / CS2 + quu);
    double hneq = L->w[i] * (qneq + cdu / CS2);
    double Si = (1.0 - 0.5 * omega) * L->w[i] * ((cF - uF) / CS2 + cu * cF / (CS2 * CS2));
    return heq + (1.0 - omega) * hneq + Si;
}

/* all directions of hprime_forced for one node (pins of the forcing term) */
int lbwp_oracle_reconstruct_forced(int lattice, const double *H10, double omega, const double *F3, double *h_out) {
    lattice_t L;
    if (lattice_make(lattice, &L)) return -1;
    for (int i = 0; i < L.q; ++i) h_out[i] = hprime_forced(&L, i, H10[0], H10 + 1, H10 + 4, omega, F3);
    return L.q;
}

/* two-component step with the near-contact force: step_2c with hprime_forced */
static void step_2c_nc(const lattice_t *L, int nx, int ny, int nz, double omega, double A, double beta,
                       double A_h, double h_c, const double *src, double *dst, double *grad, double *force) {
    const size_t n = (size_t)nx * ny * nz;
    colour_gradient(L, nx, ny, nz, src, src + n, grad);
    contact_force(L, nx, ny, nz, grad, A_h, h_c, force);
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double rA = 0.0, rB = 0.0, j[3] = {0, 0, 0}, P[6] = {0, 0, 0, 0, 0, 0};
                for (int i = 0; i < L->q; ++i) {
                    const int *c = L->c[i];
                    size_t yy = ((size_t)wrap(z - c[2], nz) * ny + wrap(y - c[1], ny)) * nx +
                                wrap(x - c[0], nx);
                    double u[3], Pn[6], G[3], F[3];
                    double a_ = src[yy], b_ = src[n + yy];
                    for (int a = 0; a < 3; ++a) u[a] = src[(2 + a) * n + yy];
                    for (int k = 0; k < 6; ++k) Pn[k] = src[(5 + k) * n + yy];
                    for (int a = 0; a < 3; ++a) G[a] = grad[a * n + yy];
                    for (int a = 0; a < 3; ++a) F[a] = force[a * n + yy];
                    double hp = hprime_forced(L, i, a_ + b_, u, Pn, omega, F);
                    double hA, hB;
                    colour_ops(L, i, hp, a_, b_, G, A, beta, &hA, &hB);
                    double hpp = hA + hB;
                    rA += hA;
                    rB += hB;
                    for (int a = 0; a < 3; ++a) j[a] += hpp * c[a];
                    for (int a = 0; a < 3; ++a)
                        for (int b = a; b < 3; ++b) P[PIDX[a][b]] += hpp * c[a] * c[b];
                }
                size_t xx = ((size_t)z * ny + y) * nx + x;
                dst[xx] = rA;
                dst[n + xx] = rB;
                for (int a = 0; a < 3; ++a) dst[(2 + a) * n + xx] = j[a] / (rA + rB);
                for (int k = 0; k < 6; ++k) dst[(5 + k) * n + xx] = P[k];
            }
}

/* Two-component run with the near-contact force; force_out (3*n doubles or NULL) receives the force field of the
 * LAST step taken (diagnostic: the pins integrate it). */
int lbwp_oracle_run_nc(int lattice, int nx, int ny, int nz, double tau, double A, double beta, double A_h,
                       double h_c, double *moments, int64_t nsteps, double *force_out) {
    lattice_t L;
    if (lattice_make(lattice, &L)) return -1;
    if (nx < 1 || ny < 1 || nz < 1 || !(tau > 0.5) || nsteps < 0 || !(h_c >= 0.0)) return -1;
    const size_t n = (size_t)nx * ny * nz;
    double *buf = (double *)malloc(sizeof(double) * 11 * n);
    double *grad = (double *)malloc(sizeof(double) * 4 * n);
    double *force = (double *)calloc(3 * n, sizeof(double));
    if (!buf || !grad || !force) { free(buf); free(grad); free(force); return -2; }
    double *cur = moments, *nxt = buf;
    for (int64_t t = 0; t < nsteps; ++t) {
        step_2c_nc(&L, nx, ny, nz, 1.0 / tau, A, beta, A_h, h_c, cur, nxt, grad, force);
        double *tmp = cur; cur = nxt; nxt = tmp;
    }
    if (cur != moments) memcpy(moments, cur, sizeof(double) * 11 * n);
    if (force_out) memcpy(force_out, force, sizeof(double) * 3 * n);
    free(buf); free(grad); free(force);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Public entry: advance `moments` (M*n doubles, layout above) by nsteps,    */
/* in place, with internal ping-pong ("Flip-Flop").              */
/* omega = 1/tau (reading C3).  Returns 0, or -1 on bad arguments / -2 on    */
/* allocation failure.                                                       */
/* ------------------------------------------------------------------------ */
int lbwp_oracle_run(int lattice, int ncomp, int nx, int ny, int nz, double tau, double A,
                    double beta, double *moments, int64_t nsteps) {
    lattice_t L;
    if (lattice_make(lattice, &L)) return -1;
    if ((ncomp != 1 && ncomp != 2) || nx < 1 || ny < 1 || nz < 1 || !(tau > 0.5) || nsteps < 0)
        return -1;
    const size_t n = (size_t)nx * ny * nz;
    const int M = ncomp == 1 ? 10 : 11;
    double *buf = (double *)malloc(sizeof(double) * M * n);
    double *grad = ncomp == 2 ? (double *)malloc(sizeof(double) * 4 * n) : NULL;
    if (!buf || (ncomp == 2 && !grad)) {
        free(buf);
        free(grad);
        return -2;
    }
    double *cur = moments, *nxt = buf;
    for (int64_t t = 0; t < nsteps; ++t) {
        if (ncomp == 1)
            step_1c(&L, nx, ny, nz, 1.0 / tau, cur, nxt);
        else
            step_2c(&L, nx, ny, nz, 1.0 / tau, A, beta, cur, nxt, grad);
        double *tmp = cur;
        cur = nxt;
        nxt = tmp;
    }
    if (cur != moments) memcpy(moments, cur, sizeof(double) * M * n);
    free(buf);
    free(grad);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* The paper's diagnostics: colour masses, total momentum, */
/* <rho>_{rho > threshold} with its node count, the maximum density, and the */
/* densities at probe sites; "rho" = density of the first component          */
/* (its field ranges from 0 to 1).  out[8] = massA, massB,     */
/* jx, jy, jz, mean above, count above, max.                                 */
/* ------------------------------------------------------------------------ */
int lbwp_oracle_diagnostics(int ncomp, int nx, int ny, int nz, const double *moments, double threshold,
                            int nprobes, const int *probe_xyz, double *out, double *probe_rho) {
    if ((ncomp != 1 && ncomp != 2) || nx < 1 || ny < 1 || nz < 1 || nprobes < 0) return -1;
    const size_t n = (size_t)nx * ny * nz;
    const int off = ncomp - 1;
    double ma = 0.0, mb = 0.0, j[3] = {0, 0, 0}, above = 0.0, count = 0.0, mx = -1e300;
    for (size_t p = 0; p < n; ++p) {
        const double ra = moments[p], rb = ncomp == 2 ? moments[n + p] : 0.0;
        ma += ra;
        mb += rb;
        for (int a = 0; a < 3; ++a) j[a] += (ra + rb) * moments[(off + 1 + a) * n + p];
        if (ra > threshold) { above += ra; count += 1.0; }
        if (ra > mx) mx = ra;
    }
    out[0] = ma; out[1] = mb; out[2] = j[0]; out[3] = j[1]; out[4] = j[2];
    out[5] = count > 0.0 ? above / count : 0.0;
    out[6] = count;
    out[7] = mx;
    for (int q = 0; q < nprobes; ++q) {
        const int x = probe_xyz[3 * q], y = probe_xyz[3 * q + 1], z = probe_xyz[3 * q + 2];
        if (x < 0 || x >= nx || y < 0 || y >= ny || z < 0 || z >= nz) return -1;
        probe_rho[q] = moments[((size_t)z * ny + y) * nx + x];
    }
    return 0;
}

int lbwp_oracle_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* number of threads the z loops use from now on (timing only: the results do not depend on it); returns what is set */
int lbwp_oracle_set_threads(int n) {
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}

/* ------------------------------------------------------------------------ */
/* Mini-oracle of the COMPARISON kernel (standard LB "with populations",     */
/* PAPER.md:29, 75, 163): two-lattice pull BGK on stored populations,        */
/*   f_i(x,t+1) = f_i(y,t) - omega [ f_i(y,t) - f_i^eq(rho(y),u(y)) ],        */
/*   y = x - c_i, f^eq = Eq. 5.  Initial f = Eq. 4 from the input moments;   */
/* output = Eq. 1-3 of the final populations.  Two components: one set of    */
/* populations per colour ("38 populations per each fluid        */
/* component"); BGK on the total, then the same perturbation and recolouring */
/* (reading C6), each colour streamed.  Initial colour split fA = rhoA/rho f.*/
/* ------------------------------------------------------------------------ */
static void pop_collide_node(const lattice_t *L, int ncomp, double omega, double A, double beta,
                             const double *fA, const double *fB, const double G[3], double *oA,
                             double *oB) {
    double f[27], H[10];
    double rA = 0.0, rB = 0.0;
    for (int i = 0; i < L->q; ++i) {
        f[i] = fA[i] + (ncomp == 2 ? fB[i] : 0.0);
        rA += fA[i];
        if (ncomp == 2) rB += fB[i];
    }
    double rho = 0.0, j[3] = {0, 0, 0};
    for (int i = 0; i < L->q; ++i) {
        rho += f[i];
        for (int a = 0; a < 3; ++a) j[a] += f[i] * L->c[i][a];
    }
    H[0] = rho;
    for (int a = 0; a < 3; ++a) H[1 + a] = j[a] / rho;
    /* P = P^eq makes hprime() return exactly Eq. 5 */
    for (int a = 0; a < 3; ++a)
        for (int b = a; b < 3; ++b)
            H[4 + PIDX[a][b]] = rho * H[1 + a] * H[1 + b] + (a == b ? rho * CS2 : 0.0);
    for (int i = 0; i < L->q; ++i) {
        double feq = hprime(L, i, H[0], H + 1, H + 4, 1.0);
        double fp = f[i] - omega * (f[i] - feq);
        if (ncomp == 1) {
            oA[i] = fp;
        } else {
            colour_ops(L, i, fp, rA, rB, G, A, beta, &oA[i], &oB[i]);
        }
    }
}

int lbwp_oracle_pop_run(int lattice, int ncomp, int nx, int ny, int nz, double tau, double A,
                        double beta, double *moments, int64_t nsteps) {
    lattice_t L;
    if (lattice_make(lattice, &L)) return -1;
    if ((ncomp != 1 && ncomp != 2) || nx < 1 || ny < 1 || nz < 1 || !(tau > 0.5) || nsteps < 0)
        return -1;
    const size_t n = (size_t)nx * ny * nz;
    const int Q = L.q, off = ncomp - 1;
    const double omega = 1.0 / tau;
    /* AoS populations [node][comp][Q]: post-collision scratch and streamed state */
    double *f = (double *)malloc(sizeof(double) * n * ncomp * Q);
    double *fc = (double *)malloc(sizeof(double) * n * ncomp * Q);
    double *rhoAB = (double *)malloc(sizeof(double) * 2 * n);
    double *grad = (double *)malloc(sizeof(double) * 4 * n);
    if (!f || !fc || !rhoAB || !grad) {
        free(f); free(fc); free(rhoAB); free(grad);
        return -2;
    }
    for (size_t p = 0; p < n; ++p) { /* initial populations: Eq. 4 (omega = 0) */
        double H[10];
        double rA = moments[p], rB = ncomp == 2 ? moments[n + p] : 0.0;
        H[0] = rA + rB;
        for (int k = 1; k < 10; ++k) H[k] = moments[(off + k) * n + p];
        for (int i = 0; i < Q; ++i) {
            double h = hprime(&L, i, H[0], H + 1, H + 4, 0.0);
            f[(p * ncomp) * Q + i] = h * (rA / H[0]);
            if (ncomp == 2) f[(p * ncomp + 1) * Q + i] = h * (rB / H[0]);
        }
    }
    for (int64_t t = 0; t < nsteps; ++t) {
        if (ncomp == 2) {
            for (size_t p = 0; p < n; ++p) {
                double a = 0.0, b = 0.0;
                for (int i = 0; i < Q; ++i) {
                    a += f[(p * 2) * Q + i];
                    b += f[(p * 2 + 1) * Q + i];
                }
                rhoAB[p] = a;
                rhoAB[n + p] = b;
            }
            colour_gradient(&L, nx, ny, nz, rhoAB, rhoAB + n, grad);
        }
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < n; ++p) { /* collide every node */
            double G[3] = {0, 0, 0};
            if (ncomp == 2)
                for (int a = 0; a < 3; ++a) G[a] = grad[a * n + p];
            pop_collide_node(&L, ncomp, omega, A, beta, &f[(p * ncomp) * Q],
                             &f[(p * ncomp + (ncomp - 1)) * Q], G, &fc[(p * ncomp) * Q],
                             &fc[(p * ncomp + (ncomp - 1)) * Q]);
        }
#pragma omp parallel for schedule(static)
        for (int z = 0; z < nz; ++z) /* pull-stream */
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    size_t xx = ((size_t)z * ny + y) * nx + x;
                    for (int i = 0; i < Q; ++i) {
                        const int *c = L.c[i];
                        size_t yy = ((size_t)wrap(z - c[2], nz) * ny + wrap(y - c[1], ny)) * nx +
                                    wrap(x - c[0], nx);
                        for (int k = 0; k < ncomp; ++k)
                            f[(xx * ncomp + k) * Q + i] = fc[(yy * ncomp + k) * Q + i];
                    }
                }
    }
    for (size_t p = 0; p < n; ++p) { /* Eq. 1-3 */
        double ft[27], H[10], rA = 0.0, rB = 0.0;
        for (int i = 0; i < Q; ++i) {
            double a = f[(p * ncomp) * Q + i];
            double b = ncomp == 2 ? f[(p * ncomp + 1) * Q + i] : 0.0;
            ft[i] = a + b;
            rA += a;
            rB += b;
        }
        lbwp_oracle_project(lattice, ft, H);
        moments[p] = rA;
        if (ncomp == 2) moments[n + p] = rB;
        for (int k = 1; k < 10; ++k) moments[(off + k) * n + p] = H[k];
    }
    free(f); free(fc); free(rhoAB); free(grad);
    return 0;
}
