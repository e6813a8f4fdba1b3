/*
 * oracle/fe_oracle.c  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU evaluation of the grand potential Omega(Delta; q, h, T)
 * of PAPER.md (arXiv 1412.8754) Eq. 5 with the quasiparticle energies of Eq. 4, for the
 * one-band, the two-band (Appendix A) and the three-band (Appendix B, numerically diagonalised) models, in the
 * loop order of Algorithm 1.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this.  It shares NO code, header, table or constant with the CUDA path under
 * paper_1412_8754_b200/csrc (it has its own parameter struct on purpose).
 *
 * What it computes (every function cites the passage it follows):
 *
 *   Omega(q, h, Delta) = sum_{eps in bands} sum_{k in grid} w_{eps k}  +  cond_mult * N^2 * Delta^2 / U
 *   w_{eps k} = f(E+) + f(E-) + C_{eps k},     f(x) = -T ln(1 + exp(-x/T))          (Eq. 5)
 *   E+- = (a - b)/2 +- sqrt(((a + b)/2)^2 + (Delta eta_k)^2)                         (Eq. 4)
 *   a = E_{eps,k} - mu - h  (spin up),  b = E_{eps,-k+q} - mu + h  (spin down)
 *   C = b (const_mode 0, reading G2)  or  E_{eps,k} - mu + h (const_mode 1, Eq. 5 literal)
 *   k = 2 pi (i, j) / N, i, j = 0..N-1                                               (reading G5)
 *
 * Every transcendental is a direct libm call at the real angle / argument; there is no
 * blocking, fusion, algebraic reuse (no cosh form, no h/Delta separation) and no reordering
 * beyond what Algorithm 1 states: line 2 "generate matrices E_{k,up} and E_{-k+q,down} for
 * k in FBZ" (tables per (q, h)), line 3 loop over Delta, lines 4-5 Eq. 4 and Eq. 5 for all k.
 * The k-sum is accumulated in long double with Neumaier compensation and rounded once to
 * fp64, so the result does not depend on summation order to ~1 ulp (reading G12).
 * f(x) is evaluated as min(x,0) - T*log1p(exp(-|x|/T)) because the literal form overflows
 * for x < -709 T (reading G7) -- same function, stable evaluation.
 *
 * The OpenMP pragma parallelises the loop over Delta, the paper's own CPU axis
 * ("parallelize the execution of the serial loop over Delta with OpenMP").
 *
 * Pins (tests/test_oracle_pins.py): Delta=0 normal state, atomic limit, -16t/pi^2, symmetries,
 * q=h=0 BCS, gap-equation stationarity, 4x4 real-space BdG brute force, two-band 4x4 orbital
 * BdG, filling n=2 at mu=1.54, pocket signs, T->0.  No function
 * here is "parity unpinned".
 *
 * Build: see oracle/build.py  (gcc -O2 -ffp-contract=off -fopenmp, no -ffast-math).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

typedef struct {
    int32_t model;       /* 1: one band  E = -2 t[0] (cos kx + cos ky)   2: two-band, Appendix A
                            3: three-band, Appendix B (hoppings in tb3, t[] unused)                */
    int32_t form_factor; /* 0: eta = eta_scale      1: eta = eta_scale cos kx cos ky */
    double  t[4];
    double  mu;
    double  U;
    double  eta_scale;
    double  cond_mult;
    int32_t band_mask;   /* bit 0: band "+" (A.4 upper sign, electron-like), bit 1: band "-"      */
    int32_t const_mode;
    double  tb3[13];     /* model 3: t1..t12 (tb3[0..11]) and eps0 (tb3[12]) of PAPER.md:242-273        */
} feo_params;

int feo_num_bands(const feo_params* p) { return p->model == 1 ? 1 : (p->model == 2 ? 2 : 3); }

int feo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void feo_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Three-band orbital Hamiltonian T_k^{alpha beta} of PAPER.md:242-270, Eqs. B.1-B.6 (row-major 3x3, real and
 * imaginary parts).  T^{12} = T^{21} real; T^{13}, T^{23} purely imaginary with T^{31} = conj(T^{13}) etc.
 * (the equation printed twice / the missing label "B.4" are reading G14 of DESIGN.md).                          */
void feo_three_band_matrix(const feo_params* p, double kx, double ky, double* re, double* im) {
    const double* t = p->tb3;              /* t[i-1] = t_i */
    const double e0 = p->tb3[12];
    for (int i = 0; i < 9; ++i) { re[i] = 0.0; im[i] = 0.0; }
    re[0] = 2.0 * t[1] * cos(kx) + 2.0 * t[0] * cos(ky) + 4.0 * t[2] * cos(kx) * cos(ky)
          + 2.0 * t[10] * (cos(2.0 * kx) - cos(2.0 * ky)) + 4.0 * t[11] * cos(2.0 * kx) * cos(2.0 * ky);   /* B.1 */
    re[4] = 2.0 * t[0] * cos(kx) + 2.0 * t[1] * cos(ky) + 4.0 * t[2] * cos(kx) * cos(ky)
          - 2.0 * t[10] * (cos(2.0 * kx) - cos(2.0 * ky)) + 4.0 * t[11] * cos(2.0 * kx) * cos(2.0 * ky);   /* B.2 */
    re[8] = e0 + 2.0 * t[4] * (cos(kx) + cos(ky)) + 4.0 * t[5] * cos(kx) * cos(ky)
          + 2.0 * t[8] * (cos(2.0 * kx) + cos(2.0 * ky))
          + 4.0 * t[9] * (cos(2.0 * kx) * cos(ky) + cos(kx) * cos(2.0 * ky));                              /* B.3 */
    re[1] = re[3] = 4.0 * t[3] * sin(kx) * sin(ky);                                                        /* B.4 */
    im[2] = 2.0 * t[6] * sin(kx) + 4.0 * t[7] * sin(kx) * cos(ky);   im[6] = -im[2];                       /* B.5 */
    im[5] = 2.0 * t[6] * sin(ky) + 4.0 * t[7] * sin(ky) * cos(kx);   im[7] = -im[5];                       /* B.6 */
}

/* Eigenvalues of a 3x3 complex Hermitian matrix (row-major re/im), ascending: the numerical band diagonalisation
 * of PAPER.md:127 ("has to be determined numerically, e.g. using ... Lapack"), Eq. 2.
 * Cyclic complex Jacobi: for each off-diagonal pair (p, q) the unitary V = diag-phase x plane rotation that zeroes
 * A[p][q] is formed explicitly and A <- V^H A V is computed by plain triple loops; sweeps repeat until the
 * off-diagonal norm is below 1e-20 of the diagonal scale (at most 60).  Pinned against LAPACK zheev (numpy eigvalsh). */
void feo_herm3_eigvals(const double* re_in, const double* im_in, double* E) {
    double ar[3][3], ai[3][3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { ar[i][j] = re_in[3 * i + j]; ai[i][j] = im_in[3 * i + j]; }
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = 0.0, diag = 0.0;
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
            const double m2 = ar[i][j] * ar[i][j] + ai[i][j] * ai[i][j];
            if (i == j) diag += m2; else off += m2;
        }
        if (off <= 1e-40 * diag || off == 0.0) break;          /* |off| <= 1e-20 |diag| */
        for (int p = 0; p < 2; ++p) for (int q = p + 1; q < 3; ++q) {
            const double beta = hypot(ar[p][q], ai[p][q]);
            if (beta == 0.0) continue;
            /* A[p][q] = beta e^{i phi}.  With P = diag(.., 1_p, .., e^{-i phi}_q, ..) the (p,q) block of P^H A P is the
             * real symmetric [[app, beta], [beta, aqq]]; the rotation J = [[c, s], [-s, c]] with
             * t = tan(theta) = sgn(tau) / (|tau| + sqrt(1 + tau^2)), tau = (aqq - app) / (2 beta) diagonalises it. */
            const double cphi = ar[p][q] / beta, sphi = ai[p][q] / beta;
            const double tau = (ar[q][q] - ar[p][p]) / (2.0 * beta);
            const double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
            const double c = 1.0 / sqrt(1.0 + t * t), s = t * c;
            double vr[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}}, vi[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
            /* V = P J :  V[p][p] = c, V[p][q] = s, V[q][p] = -s e^{-i phi}, V[q][q] = c e^{-i phi} */
            vr[p][p] = c;          vi[p][p] = 0.0;
            vr[p][q] = s;          vi[p][q] = 0.0;
            vr[q][p] = -s * cphi;  vi[q][p] = s * sphi;
            vr[q][q] = c * cphi;   vi[q][q] = -c * sphi;
            double br[3][3], bi[3][3], cr[3][3], ci[3][3];
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {          /* B = A V */
                double xr = 0.0, xi = 0.0;
                for (int k = 0; k < 3; ++k) {
                    xr += ar[i][k] * vr[k][j] - ai[i][k] * vi[k][j];
                    xi += ar[i][k] * vi[k][j] + ai[i][k] * vr[k][j];
                }
                br[i][j] = xr; bi[i][j] = xi;
            }
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {          /* C = V^H B */
                double xr = 0.0, xi = 0.0;
                for (int k = 0; k < 3; ++k) {
                    xr += vr[k][i] * br[k][j] + vi[k][i] * bi[k][j];
                    xi += vr[k][i] * bi[k][j] - vi[k][i] * br[k][j];
                }
                cr[i][j] = xr; ci[i][j] = xi;
            }
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { ar[i][j] = cr[i][j]; ai[i][j] = ci[i][j]; }
            for (int i = 0; i < 3; ++i) ai[i][i] = 0.0;
            ar[p][q] = ar[q][p] = 0.0; ai[p][q] = ai[q][p] = 0.0;   /* zero by construction; drop the rounding residue */
        }
    }
    double e0 = ar[0][0], e1 = ar[1][1], e2 = ar[2][2], tmp;
    if (e0 > e1) { tmp = e0; e0 = e1; e1 = tmp; }
    if (e1 > e2) { tmp = e1; e1 = e2; e2 = tmp; }
    if (e0 > e1) { tmp = e0; e0 = e1; e1 = tmp; }
    E[0] = e0; E[1] = e1; E[2] = e2;
}

/* Band energies E_{eps,k} WITHOUT the -(mu + sigma h) shift.
 * one band: nearest-neighbour square lattice (BASELINE.json config 1; reading G13).
 * two band: PAPER.md:216-227, Eqs. A.1-A.4; E[0] = E_+ (electron-like), E[1] = E_- (hole-like).
 * three band: eigenvalues of B.1-B.6 in ascending order, E[0] <= E[1] <= E[2] (reading G18).  */
void feo_band_energies(const feo_params* p, double kx, double ky, double* E) {
    if (p->model == 1) {
        E[0] = -2.0 * p->t[0] * (cos(kx) + cos(ky));
        return;
    }
    if (p->model == 3) {
        double re[9], im[9];
        feo_three_band_matrix(p, kx, ky, re, im);
        feo_herm3_eigvals(re, im, E);
        return;
    }
    const double t1 = p->t[0], t2 = p->t[1], t3 = p->t[2], t4 = p->t[3];
    const double T11 = -2.0 * (t1 * cos(kx) + t2 * cos(ky)) - 4.0 * t3 * cos(kx) * cos(ky); /* A.1 */
    const double T22 = -2.0 * (t2 * cos(kx) + t1 * cos(ky)) - 4.0 * t3 * cos(kx) * cos(ky); /* A.2 */
    const double T12 = -4.0 * t4 * sin(kx) * sin(ky);                                       /* A.3 */
    const double avg = (T11 + T22) / 2.0;
    const double rad = sqrt(((T11 - T22) / 2.0) * ((T11 - T22) / 2.0) + T12 * T12);
    E[0] = avg + rad;                                                                       /* A.4 */
    E[1] = avg - rad;
}

/* Form factor eta(k): PAPER.md:53 ("proportional to cos kx cos ky"), :87; normalisation = reading G4. */
double feo_eta(const feo_params* p, double kx, double ky) {
    if (p->form_factor == 0) return p->eta_scale;
    return p->eta_scale * cos(kx) * cos(ky);
}

/* Eq. 4: a = E_{k,up} (shifted), b = E_{-k+q,down} (shifted), gap = Delta*eta(k). */
void feo_quasiparticle(double a, double b, double gap, double* Eplus, double* Eminus) {
    const double half_diff = (a - b) / 2.0;
    const double half_sum  = (a + b) / 2.0;
    const double root = sqrt(half_sum * half_sum + gap * gap);
    *Eplus  = half_diff + root;
    *Eminus = half_diff - root;
}

/* f(x) = -(1/beta) ln(1 + exp(-beta x)), the summand of Eq. 5's first term. */
double feo_thermal(double x, double T) {
    const double neg = x < 0.0 ? x : 0.0;
    return neg - T * log1p(exp(-fabs(x) / T));
}

typedef struct { long double s, c; } feo_acc;   /* Neumaier compensated accumulator */
static inline void acc_add(feo_acc* A, long double x) {
    const long double t = A->s + x;
    if (fabsl(A->s) >= fabsl(x)) A->c += (A->s - t) + x;
    else                         A->c += (x - t) + A->s;
    A->s = t;
}

/*
 * One (q, h) column of Algorithm 1: line 2 builds the tables, lines 3-7
 * loop over Delta.  omega_out[id] = Omega(q, h, delta[id]).   Returns 0, or -1 on bad input,
 * -2 on allocation failure.
 */
int feo_omega_column(const feo_params* p, int32_t N, double T, double qx, double qy, double h,
                     const double* delta, int32_t nd, double* omega_out) {
    if (!p || !delta || !omega_out || N < 1 || nd < 1 || !(T > 0.0) || !(p->U > 0.0)) return -1;
    if (p->model != 1 && p->model != 2 && p->model != 3) return -1;
    const int nb = feo_num_bands(p);
    const size_t nk = (size_t)N * (size_t)N;
    double* up  = (double*)malloc(sizeof(double) * nk * nb);   /* xi_{eps,k,up}        */
    double* dn  = (double*)malloc(sizeof(double) * nk * nb);   /* xi_{eps,-k+q,down}   */
    double* cst = (double*)malloc(sizeof(double) * nk * nb);   /* constant term of Eq. 5 */
    double* eta = (double*)malloc(sizeof(double) * nk);
    if (!up || !dn || !cst || !eta) { free(up); free(dn); free(cst); free(eta); return -2; }

    /* Algorithm 1 line 2: "generate matrices E_{eps k up} and E_{eps,-k+q,down} for k in FBZ". */
#pragma omp parallel for schedule(static)
    for (int32_t j = 0; j < N; ++j) {
        for (int32_t i = 0; i < N; ++i) {
            const double kx = 2.0 * M_PI * (double)i / (double)N;
            const double ky = 2.0 * M_PI * (double)j / (double)N;
            double Ek[3], Ekq[3];
            feo_band_energies(p, kx, ky, Ek);
            feo_band_energies(p, -kx + qx, -ky + qy, Ekq);
            const size_t k = (size_t)j * N + i;
            eta[k] = feo_eta(p, kx, ky);
            for (int e = 0; e < nb; ++e) {
                up[e * nk + k]  = Ek[e]  - p->mu - h;     /* sigma = up   = +1 (reading G1) */
                dn[e * nk + k]  = Ekq[e] - p->mu + h;     /* sigma = down = -1              */
                cst[e * nk + k] = (p->const_mode == 0) ? dn[e * nk + k] : (Ek[e] - p->mu + h);
            }
        }
    }

    /* Algorithm 1 lines 3-7: for Delta = 0..Delta_max: Eq. 4 for all k, then Omega (Eq. 5). */
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t id = 0; id < nd; ++id) {
        const double D = delta[id];
        feo_acc A = {0.0L, 0.0L};
        for (int e = 0; e < nb; ++e) {
            if (!((p->band_mask >> e) & 1)) continue;
            for (size_t k = 0; k < nk; ++k) {
                double Ep, Em;
                feo_quasiparticle(up[e * nk + k], dn[e * nk + k], D * eta[k], &Ep, &Em);
                acc_add(&A, (long double)feo_thermal(Ep, T));
                acc_add(&A, (long double)feo_thermal(Em, T));
                acc_add(&A, (long double)cst[e * nk + k]);
            }
        }
        /* condensation term: -2|Delta|^2/V per band per k in Eq. 5 == +cond_mult N^2 Delta^2/U (reading G3) */
        acc_add(&A, (long double)p->cond_mult * (long double)nk * (long double)D * (long double)D
                        / (long double)p->U);
        omega_out[id] = (double)(A.s + A.c);
    }
    free(up); free(dn); free(cst); free(eta);
    return 0;
}

/*
 * Diagnostic for the parity tests (not a step of the method): the MAGNITUDE of the sum feo_omega_column forms,
 *   mag_out[id] = sum_{eps, k} ( |f(E+)| + |f(E-)| + |C_{eps k}| ) + |condensation term|,
 * i.e. the same terms of Eq. 5 with absolute values.  mag / |Omega| is the condition number of the
 * k-sum: where the terms cancel (a single, nearly empty band selected by band_mask) no fp64 evaluation can be
 * accurate to 1e-12 of |Omega| itself, and the tests bound the error by the rounding of the terms instead.
 */
int feo_omega_column_magnitude(const feo_params* p, int32_t N, double T, double qx, double qy, double h,
                               const double* delta, int32_t nd, double* mag_out) {
    if (!p || !delta || !mag_out || N < 1 || nd < 1 || !(T > 0.0) || !(p->U > 0.0)) return -1;
    if (p->model != 1 && p->model != 2 && p->model != 3) return -1;
    const int nb = feo_num_bands(p);
    const size_t nk = (size_t)N * (size_t)N;
    double* up  = (double*)malloc(sizeof(double) * nk * nb);
    double* dn  = (double*)malloc(sizeof(double) * nk * nb);
    double* cst = (double*)malloc(sizeof(double) * nk * nb);
    double* eta = (double*)malloc(sizeof(double) * nk);
    if (!up || !dn || !cst || !eta) { free(up); free(dn); free(cst); free(eta); return -2; }
#pragma omp parallel for schedule(static)
    for (int32_t j = 0; j < N; ++j)
        for (int32_t i = 0; i < N; ++i) {
            const double kx = 2.0 * M_PI * (double)i / (double)N;
            const double ky = 2.0 * M_PI * (double)j / (double)N;
            double Ek[3], Ekq[3];
            feo_band_energies(p, kx, ky, Ek);
            feo_band_energies(p, -kx + qx, -ky + qy, Ekq);
            const size_t k = (size_t)j * N + i;
            eta[k] = feo_eta(p, kx, ky);
            for (int e = 0; e < nb; ++e) {
                up[e * nk + k]  = Ek[e]  - p->mu - h;
                dn[e * nk + k]  = Ekq[e] - p->mu + h;
                cst[e * nk + k] = (p->const_mode == 0) ? dn[e * nk + k] : (Ek[e] - p->mu + h);
            }
        }
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t id = 0; id < nd; ++id) {
        const double D = delta[id];
        feo_acc A = {0.0L, 0.0L};
        for (int e = 0; e < nb; ++e) {
            if (!((p->band_mask >> e) & 1)) continue;
            for (size_t k = 0; k < nk; ++k) {
                double Ep, Em;
                feo_quasiparticle(up[e * nk + k], dn[e * nk + k], D * eta[k], &Ep, &Em);
                acc_add(&A, fabsl((long double)feo_thermal(Ep, T)));
                acc_add(&A, fabsl((long double)feo_thermal(Em, T)));
                acc_add(&A, fabsl((long double)cst[e * nk + k]));
            }
        }
        acc_add(&A, fabsl((long double)p->cond_mult * (long double)nk * (long double)D * (long double)D
                          / (long double)p->U));
        mag_out[id] = (double)(A.s + A.c);
    }
    free(up); free(dn); free(cst); free(eta);
    return 0;
}

/* Whole grid, Algorithm 1's outer loops: q, then h, then the column above.
 * omega_out index (iq*nh + ih)*nd + id  (Delta fastest).                                      */
int feo_omega_grid(const feo_params* p, int32_t N, double T,
                   const double* q_xy, int32_t nq, const double* h, int32_t nh,
                   const double* delta, int32_t nd, double* omega_out) {
    if (!q_xy || !h || nq < 1 || nh < 1) return -1;
    for (int32_t iq = 0; iq < nq; ++iq)
        for (int32_t ih = 0; ih < nh; ++ih) {
            int rc = feo_omega_column(p, N, T, q_xy[2 * iq], q_xy[2 * iq + 1], h[ih], delta, nd,
                                      omega_out + ((size_t)iq * nh + ih) * nd);
            if (rc) return rc;
        }
    return 0;
}

/* Algorithm 1 line 6 / step 3 of PAPER.md:169: linear search for the lowest Omega over Delta,
 * strict '<' so the lowest index wins among exact ties (reading G11).                          */
int feo_argmin(const double* omega, const double* delta, int32_t ncol, int32_t nd,
               int32_t* idx_out, double* delta_star, double* omega_star) {
    if (!omega || !delta || ncol < 1 || nd < 1) return -1;
    for (int32_t c = 0; c < ncol; ++c) {
        int32_t best = 0;
        for (int32_t id = 1; id < nd; ++id)
            if (omega[(size_t)c * nd + id] < omega[(size_t)c * nd + best]) best = id;
        if (idx_out)    idx_out[c] = best;
        if (delta_star) delta_star[c] = delta[best];
        if (omega_star) omega_star[c] = omega[(size_t)c * nd + best];
    }
    return 0;
}

/* Outer loops of Algorithm 1: for a fixed field h the global ground state is
 * the (q, Delta) pair of lowest Omega: "Omega_0 := +inf; for q: for Delta: if Omega < Omega_0 then save".
 * omega is the grid of feo_omega_grid, index (iq*nh + ih)*nd + id.  ref_id >= 0: the value compared across q is the
 * condensation energy Omega(q, h, Delta) - Omega(q, h, delta[ref_id]) (reading G17: for off-grid q the
 * normal-state Omega itself depends on q at finite N); ref_id = -1: Omega itself, Algorithm 1 as printed.
 * Strict '<' in loop order q, then Delta: the lowest (iq, id) wins among exact ties.                            */
int feo_argmin_q(const double* omega, int32_t nq, int32_t nh, int32_t nd, int32_t ref_id,
                 int32_t* iq_out, int32_t* id_out, double* value_out) {
    if (!omega || nq < 1 || nh < 1 || nd < 1 || ref_id < -1 || ref_id >= nd) return -1;
    for (int32_t ih = 0; ih < nh; ++ih) {
        double best = INFINITY;
        int32_t bq = 0, bd = 0;
        for (int32_t iq = 0; iq < nq; ++iq) {
            const double* col = omega + ((size_t)iq * nh + ih) * nd;
            for (int32_t id = 0; id < nd; ++id) {
                const double v = ref_id >= 0 ? col[id] - col[ref_id] : col[id];
                if (v < best) { best = v; bq = iq; bd = id; }
            }
        }
        if (iq_out) iq_out[ih] = bq;
        if (id_out) id_out[ih] = bd;
        if (value_out) value_out[ih] = best;
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------------------
 * Static Cooper-pair susceptibility, Appendix C, Eqs. C.2-C.3 at omega -> 0:
 *
 *   chi_{eps eps'}(q) = -(1/N) sum_k eta(-k-q)^2 [ f(-E_{eps k up}) - f(E_{eps',-k-q,down}) ] / ( -E_{eps k up} - E_{eps',-k-q,down} )
 *
 * N = number of lattice sites = number of k-points, f(x) = 1/(exp(x/T) + 1) the Fermi function, E_{eps k sigma}
 * the band energies INCLUDING -(mu + sigma h) (Eq. 2), eta(k) = eta_scale cos kx cos ky
 * (eta_scale = 4 is the paper's C.3 normalisation; reading G4).  The delta_{kl} of C.3 has been summed out.
 * feo_pair_term is the summand's thermal factor  [f(-a) - f(b)] / (a + b)  evaluated literally in long double;
 * at a + b -> 0 the quotient is 0/0 and its limit -f'((a-b)/2) = 1 / (4 T cosh^2((a-b) / 4T)) is used.
 * chi_out[(iq*nb + eps)*nb + eps'], nb = number of bands.  Returns 0, -1 bad input.
 * --------------------------------------------------------------------------------------------------------- */
static long double feo_fermi_l(long double x, long double T) { return 1.0L / (expl(x / T) + 1.0L); }

double feo_pair_term(double a, double b, double T) {
    const long double al = a, bl = b, Tl = T;
    const long double den = al + bl;
    /* Removable singularity of C.3 (reading G19): with a = m + e, b = -m + e the quotient is the central
     * difference [f(-m-e) - f(-m+e)] / (2e) = -f'(m) (1 + O((e/T)^2)); for |a + b| <= 1e-6 T the literal quotient
     * would lose its digits to cancellation (it is 0/0 at e = 0) while the limit is exact to 1e-13. */
    if (fabsl(den) <= 1e-6L * Tl) {
        const long double c = coshl((al - bl) / (4.0L * Tl));
        return (double)(1.0L / (4.0L * Tl * c * c));
    }
    return (double)((feo_fermi_l(-al, Tl) - feo_fermi_l(bl, Tl)) / den);
}

int feo_pair_susceptibility(const feo_params* p, int32_t N, double T, const double* q_xy, int32_t nq, double h,
                            double* chi_out) {
    if (!p || !q_xy || !chi_out || N < 1 || nq < 1 || !(T > 0.0)) return -1;
    if (p->model != 1 && p->model != 2 && p->model != 3) return -1;
    const int nb = feo_num_bands(p);
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t iq = 0; iq < nq; ++iq) {
        const double qx = q_xy[2 * iq], qy = q_xy[2 * iq + 1];
        feo_acc A[9];
        for (int i = 0; i < 9; ++i) { A[i].s = 0.0L; A[i].c = 0.0L; }
        for (int32_t j = 0; j < N; ++j)
            for (int32_t i = 0; i < N; ++i) {
                const double kx = 2.0 * M_PI * (double)i / (double)N;
                const double ky = 2.0 * M_PI * (double)j / (double)N;
                double Ek[3], Ekq[3];
                feo_band_energies(p, kx, ky, Ek);                    /* E_{eps}(k)     */
                feo_band_energies(p, -kx - qx, -ky - qy, Ekq);       /* E_{eps'}(-k-q) */
                const double eta = feo_eta(p, -kx - qx, -ky - qy);   /* eta(-k-q), C.2 */
                for (int e = 0; e < nb; ++e)
                    for (int f = 0; f < nb; ++f) {
                        const double a = Ek[e] - p->mu - h;          /* E_{eps k up}          */
                        const double b = Ekq[f] - p->mu + h;         /* E_{eps',-k-q,down}    */
                        acc_add(&A[e * nb + f], (long double)(eta * eta) * (long double)feo_pair_term(a, b, T));
                    }
            }
        for (int e = 0; e < nb * nb; ++e)
            chi_out[(size_t)iq * nb * nb + e] = (double)((A[e].s + A[e].c) / ((long double)N * (long double)N));
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------------------
 * Single-precision variant ("the same CUDA C code in double precision (DP), single
 * precision (SP), and single precision with fast intrinsic functions (SPFM)").
 * The same Algorithm 1 / Eq. 4 / Eq. 5 as feo_omega_column with EVERY per-term operation in IEEE binary32
 * (cosf, sinf, sqrtf, expf, log1pf; k, q, h, Delta, T, mu, hoppings rounded to float first).  Only the sum over k
 * is kept in double (compensated), so that the result does not depend on summation order and can be compared
 * (reading G20; the paper's kernel sums in float, order unspecified).  SPFM has no CPU counterpart (the
 * "fast intrinsics" are GPU instructions): the SPFM kernel is compared with this function at a wider tolerance.
 * One- and two-band models only.  Returns 0, -1 bad input, -2 allocation failure.
 * --------------------------------------------------------------------------------------------------------- */
static void feo_band_energies_sp(const feo_params* p, float kx, float ky, float* E) {
    if (p->model == 1) {
        E[0] = -2.0f * (float)p->t[0] * (cosf(kx) + cosf(ky));
        return;
    }
    const float t1 = (float)p->t[0], t2 = (float)p->t[1], t3 = (float)p->t[2], t4 = (float)p->t[3];
    const float T11 = -2.0f * (t1 * cosf(kx) + t2 * cosf(ky)) - 4.0f * t3 * cosf(kx) * cosf(ky);   /* A.1 */
    const float T22 = -2.0f * (t2 * cosf(kx) + t1 * cosf(ky)) - 4.0f * t3 * cosf(kx) * cosf(ky);   /* A.2 */
    const float T12 = -4.0f * t4 * sinf(kx) * sinf(ky);                                            /* A.3 */
    const float avg = (T11 + T22) / 2.0f;
    const float rad = sqrtf(((T11 - T22) / 2.0f) * ((T11 - T22) / 2.0f) + T12 * T12);
    E[0] = avg + rad;                                                                              /* A.4 */
    E[1] = avg - rad;
}

static float feo_thermal_sp(float x, float T) {          /* f(x) = -T ln(1 + exp(-x/T)), stable form, in float */
    const float neg = x < 0.0f ? x : 0.0f;
    return neg - T * log1pf(expf(-fabsf(x) / T));
}

int feo_omega_column_sp(const feo_params* p, int32_t N, double T, double qx, double qy, double h,
                        const double* delta, int32_t nd, double* omega_out) {
    if (!p || !delta || !omega_out || N < 1 || nd < 1 || !(T > 0.0) || !(p->U > 0.0)) return -1;
    if (p->model != 1 && p->model != 2) return -1;
    const int nb = feo_num_bands(p);
    const size_t nk = (size_t)N * (size_t)N;
    float* up  = (float*)malloc(sizeof(float) * nk * nb);
    float* dn  = (float*)malloc(sizeof(float) * nk * nb);
    float* cst = (float*)malloc(sizeof(float) * nk * nb);
    float* eta = (float*)malloc(sizeof(float) * nk);
    if (!up || !dn || !cst || !eta) { free(up); free(dn); free(cst); free(eta); return -2; }
    const float Tf = (float)T, muf = (float)p->mu, hf = (float)h, qxf = (float)qx, qyf = (float)qy;
    const float twopi = (float)(2.0 * M_PI);
    for (int32_t j = 0; j < N; ++j)
        for (int32_t i = 0; i < N; ++i) {
            const float kx = twopi * (float)i / (float)N, ky = twopi * (float)j / (float)N;
            float Ek[2], Ekq[2];
            feo_band_energies_sp(p, kx, ky, Ek);
            feo_band_energies_sp(p, -kx + qxf, -ky + qyf, Ekq);
            const size_t k = (size_t)j * N + i;
            eta[k] = p->form_factor == 0 ? (float)p->eta_scale : (float)p->eta_scale * cosf(kx) * cosf(ky);
            for (int e = 0; e < nb; ++e) {
                up[e * nk + k]  = Ek[e]  - muf - hf;
                dn[e * nk + k]  = Ekq[e] - muf + hf;
                cst[e * nk + k] = (p->const_mode == 0) ? dn[e * nk + k] : (Ek[e] - muf + hf);
            }
        }
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t id = 0; id < nd; ++id) {
        const float D = (float)delta[id];
        feo_acc A = {0.0L, 0.0L};
        for (int e = 0; e < nb; ++e) {
            if (!((p->band_mask >> e) & 1)) continue;
            for (size_t k = 0; k < nk; ++k) {
                const float a = up[e * nk + k], b = dn[e * nk + k], gap = D * eta[k];
                const float half_diff = (a - b) / 2.0f, half_sum = (a + b) / 2.0f;
                const float root = sqrtf(half_sum * half_sum + gap * gap);                 /* Eq. 4 */
                const float term = feo_thermal_sp(half_diff + root, Tf) + feo_thermal_sp(half_diff - root, Tf)
                                 + cst[e * nk + k];                                        /* Eq. 5 */
                acc_add(&A, (long double)term);
            }
        }
        acc_add(&A, (long double)p->cond_mult * (long double)nk * (long double)delta[id] * (long double)delta[id]
                        / (long double)p->U);
        omega_out[id] = (double)(A.s + A.c);
    }
    free(up); free(dn); free(cst); free(eta);
    return 0;
}
