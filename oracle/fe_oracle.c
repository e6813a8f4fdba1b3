/*
 * oracle/fe_oracle.c  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU evaluation of the grand potential Omega(Delta; q, h, T)
 * of PAPER.md (arXiv 1412.8754) Eq. 5 with the quasiparticle energies of Eq. 4, for the
 * one-band and the two-band (Appendix A) models, in the loop order of Algorithm 1.
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
    int32_t model;       /* 1: one band  E = -2 t[0] (cos kx + cos ky)   2: two-band, Appendix A  */
    int32_t form_factor; /* 0: eta = eta_scale      1: eta = eta_scale cos kx cos ky */
    double  t[4];
    double  mu;
    double  U;
    double  eta_scale;
    double  cond_mult;
    int32_t band_mask;   /* bit 0: band "+" (A.4 upper sign, electron-like), bit 1: band "-"      */
    int32_t const_mode;
} feo_params;

int feo_num_bands(const feo_params* p) { return p->model == 1 ? 1 : 2; }

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

/* Band energies E_{eps,k} WITHOUT the -(mu + sigma h) shift.
 * one band: nearest-neighbour square lattice (BASELINE.json config 1; reading G13).
 * two band: PAPER.md:216-227, Eqs. A.1-A.4; E[0] = E_+ (electron-like), E[1] = E_- (hole-like).   */
void feo_band_energies(const feo_params* p, double kx, double ky, double* E) {
    if (p->model == 1) {
        E[0] = -2.0 * p->t[0] * (cos(kx) + cos(ky));
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
    if (p->model != 1 && p->model != 2) return -1;
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
            double Ek[2], Ekq[2];
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
