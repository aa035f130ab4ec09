/*
 * oracle/aton_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the ATON hot path (explicit M1 moment radiative transfer
 * + hydrogen photo-chemistry/cooling) of Aubert & Teyssier, "Reionization simulations powered by
 * GPUs I".  It exists so that tests, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference leg can check and time the CUDA library against it.  It shares
 * no code, header, table or constant with paper_1004_2503_b200/csrc/ and nothing in the product
 * path may call it.
 *
 * Every function follows the paper's (or, where the paper is silent or garbled, DESIGN.md's
 * "Readings") statement step by step: no blocking, no fusion, no reordering.  OpenMP only splits
 * the outer z loop of per-cell work (each cell is independent).
 *
 * Units: CGS.  N [photons cm^-3], F [photons cm^-2 s^-1], n_H [cm^-3], T [K], x = n_HII/n_H.
 * Layout: C order [nz][ny][nx], x fastest; cell (i,j,k) at i + nx*(j + ny*k); periodic box.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closure limits and trace (P0), free-streaming
 * binomial (P1), vacuum conservation (P2), realizability (P3), diffusion-limit amplification
 * matrix (P4), photon budget + brute-force root of the backward-Euler system (P5), equilibrium
 * closed form (P6), Stroemgren volume (P7), first step from vacuum (P8), cube symmetry (P9),
 * textbook spot values of the rate fits (S7): alpha_A/B (3 %), z_rec (5 %), z_ff prefactor, z_exc against the
 * two-level Lyman-alpha rate (factor 2) and its Boltzmann temperature (1e-3), the Compton coefficient from CODATA
 * constants (1 %) and its sign, the 10 % rule as an inequality on every accepted sub-step, F' = c n N' on f = 1 beams.
 * LOOSEST PIN: the collisional-ionisation fit beta (and z_ci = 13.6 eV * beta) is held to 25 % of an independent
 * (different-author) closed form only; no table value is in the container to do better.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define K_BOLTZ 1.380649e-16      /* erg/K */
#define EV_ERG 1.602176634e-12    /* erg per eV */
#define E0_EV 13.6                /* H ionisation threshold, eV (SURVEY O4 "e0 = 13.6 eV") */
#define T_MIN 1.0                 /* K, reading S18 */
#define T_CMB0 2.726

typedef struct {
    double c;            /* speed of light used by the transport, cm/s */
    double dx;           /* cell size, cm */
    double sigma_n;      /* number-weighted cross-section, cm^2 */
    double sigma_e;      /* energy-weighted cross-section, cm^2 */
    double e_photon_eV;  /* mean photon energy, eV */
    double clump_a, clump_b;
    double redshift;     /* <0: no Compton cooling */
    double eps_sub;      /* sub-cycle energy tolerance (Anninos 10% rule), reading S5 */
    double nH_mean;      /* <n_H>_V used by the linear clumping law, reading S8 */
    double clump_i_a, clump_i_b; /* photo-ionisation clumping C_I = max(1, a nH^b) of Eq.15 (L247-249, L269:
                                    "C_I ~ n_H^0.2"); a <= 0: C_I = 1 (reading S8b) */
    int recomb_case;     /* 1: case B, on-the-spot; 0: case A + recombination radiation (S6) */
    int cooling;         /* 0: T frozen; 1: heating + cooling */
    int coll_ion;        /* collisional ionisation on/off */
    int clump_model;     /* 0 none; 1: C=max(1,a+b*delta); 2: C=max(1,a*nH^b) */
    int max_sub;         /* sub-cycle cap (S18) */
    int flux;            /* intercell flux: 0 Lax-Friedrichs (the one the paper used), 1 HLL */
} orc_params;

typedef struct {          /* T-dependent coefficients, reading S7 (Hui & Gnedin 1997; Cen 1992) */
    double alpha_A, alpha_B, beta;                    /* cm^3/s */
    double z_recA, z_recB, z_ci, z_exc, z_ff;         /* erg cm^3/s */
    double dl_recA, dl_recB, dl_ci, dl_exc, dl_ff;    /* d ln(zeta) / d ln T */
} orc_rates_t;

void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int orc_get_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * O1 closure.  PAPER.md:L70-78, Eq.5-6 with the I / n(x)n coefficients un-swapped (reading G1) and
 * chi(f) = (3+4f^2)/(5+2 sqrt(4-3f^2)) (reading S1: the M1 / Levermore form; chi(0)=1/3, chi(1)=1).
 * ------------------------------------------------------------------------------------------- */
double orc_chi(double f) {
    return (3.0 + 4.0 * f * f) / (5.0 + 2.0 * sqrt(4.0 - 3.0 * f * f));
}

/* P[3*a+b] = D_ab N,  D = (1-chi)/2 I + (3chi-1)/2 n(x)n,  f = min(1,|F|/(cN)), n = F/|F| (S2). */
void orc_closure(double N, const double F[3], double c, double P[9]) {
    double Fn = sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
    double f = 0.0, n[3] = {0.0, 0.0, 0.0};
    if (N > 0.0) {
        f = Fn / (c * N);
        if (f > 1.0) f = 1.0;
    }
    if (Fn > 0.0) {
        n[0] = F[0] / Fn; n[1] = F[1] / Fn; n[2] = F[2] / Fn;
    }
    double chi = orc_chi(f);
    for (int a = 0; a < 3; a++)
        for (int b = 0; b < 3; b++)
            P[3 * a + b] = (0.5 * (1.0 - chi) * (a == b ? 1.0 : 0.0)
                            + 0.5 * (3.0 * chi - 1.0) * n[a] * n[b]) * N;
}

/* ---------------------------------------------------------------------------------------------
 * O2 transport.  PAPER.md Eq.3-4 without the kappa terms, Eq.A2/A5 (L428, L447), with the
 * Lax-Friedrichs intercell flux at speed c (L85; reading S4):
 *     FF_{i+1/2} = (FF_i + FF_{i+1})/2 - (c/2)(U_{i+1} - U_i),
 * U = (N, Fx, Fy, Fz), FF_d(N) = F_d, FF_d(F_j) = c^2 P_dj.  Unsplit in 3-D, periodic, Jacobi.
 * ------------------------------------------------------------------------------------------- */
static inline long wrap(long i, long n) { return (i % n + n) % n; }

/* physical flux of the 4 conserved variables through a face normal to axis d, from cell state */
static void flux_fn(int d, double N, const double F[3], double c, double out[4]) {
    double P[9];
    orc_closure(N, F, c, P);
    out[0] = F[d];
    out[1] = c * c * P[3 * d + 0];
    out[2] = c * c * P[3 * d + 1];
    out[3] = c * c * P[3 * d + 2];
}

void orc_transport(int nx, int ny, int nz, const double *N, const double *Fx, const double *Fy,
                   const double *Fz, double c, double dx, double dt,
                   double *N1, double *Fx1, double *Fy1, double *Fz1) {
    const long sx = 1, sy = nx, sz = (long)nx * ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                long id = i * sx + j * sy + k * sz;
                double U[4] = {N[id], Fx[id], Fy[id], Fz[id]};
                double Fc[3] = {Fx[id], Fy[id], Fz[id]};
                double Un[4] = {U[0], U[1], U[2], U[3]};
                for (int d = 0; d < 3; d++) {
                    long ip, im;
                    if (d == 0) { ip = wrap(i + 1, nx) * sx + j * sy + k * sz; im = wrap(i - 1, nx) * sx + j * sy + k * sz; }
                    else if (d == 1) { ip = i * sx + wrap(j + 1, ny) * sy + k * sz; im = i * sx + wrap(j - 1, ny) * sy + k * sz; }
                    else { ip = i * sx + j * sy + wrap(k + 1, nz) * sz; im = i * sx + j * sy + wrap(k - 1, nz) * sz; }
                    double Up[4] = {N[ip], Fx[ip], Fy[ip], Fz[ip]};
                    double Um[4] = {N[im], Fx[im], Fy[im], Fz[im]};
                    double Fp[3] = {Fx[ip], Fy[ip], Fz[ip]}, Fm[3] = {Fx[im], Fy[im], Fz[im]};
                    double g0[4], gp[4], gm[4];
                    flux_fn(d, U[0], Fc, c, g0);
                    flux_fn(d, Up[0], Fp, c, gp);
                    flux_fn(d, Um[0], Fm, c, gm);
                    for (int v = 0; v < 4; v++) {
                        double f_hi = 0.5 * (g0[v] + gp[v]) - 0.5 * c * (Up[v] - U[v]);  /* i+1/2 */
                        double f_lo = 0.5 * (gm[v] + g0[v]) - 0.5 * c * (U[v] - Um[v]);  /* i-1/2 */
                        Un[v] -= dt / dx * (f_hi - f_lo);                                /* Eq.A2 */
                    }
                }
                N1[id] = Un[0]; Fx1[id] = Un[1]; Fy1[id] = Un[2]; Fz1[id] = Un[3];
            }
}

/* ---------------------------------------------------------------------------------------------
 * O2' transport with the HLL intercell flux ("the code is able to evaluate intercell fluxes using
 * both the ... HLL or the simpler Lax-Friedrich scheme"; reading S20).  The paper prints
 * neither the flux nor the wave speeds; the standard Harten-Lax-van Leer form for the M1 system is taken:
 *     FF_{i+1/2} = [ l+ FF_i - l- FF_{i+1} + l+ l- (U_{i+1} - U_i) ] / (l+ - l-),
 *     l+ = max(0, lmax_i, lmax_{i+1}),   l- = min(0, lmin_i, lmin_{i+1}),
 * with lmin, lmax the extreme eigenvalues of the Jacobian d FF_d / d U of the M1 flux function in the direction d
 * of the face.  For the Levermore closure they have the closed form (in units of c; mu = F_d/|F|, xi = sqrt(4-3f^2))
 *     l(+-) = [ mu f +- sqrt( (2/3)(xi^2 - xi) + 2 mu^2 (2 - f^2 - xi) ) ] / xi
 * (pinned in tests/test_oracle_hll.py against numpy's eigenvalues of the finite-difference Jacobian of flux_fn).
 * With l+ = -l- = c the flux is the Lax-Friedrichs flux of orc_transport.
 * ------------------------------------------------------------------------------------------- */
void orc_m1_wavespeeds(double N, const double F[3], double c, int d, double *lmin, double *lmax) {
    double Fn = sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
    double f = 0.0, mu = 0.0;
    if (N > 0.0) {
        f = Fn / (c * N);
        if (f > 1.0) f = 1.0;
    }
    if (Fn > 0.0) mu = F[d] / Fn;
    double xi = sqrt(4.0 - 3.0 * f * f);
    double disc = (2.0 / 3.0) * (xi * xi - xi) + 2.0 * mu * mu * (2.0 - f * f - xi);
    double root = sqrt(disc > 0.0 ? disc : 0.0);
    *lmin = c * (mu * f - root) / xi;
    *lmax = c * (mu * f + root) / xi;
}

/* physical flux through a face normal to axis d (the oracle's own flux_fn, exported for the Jacobian pin) */
void orc_flux_fn(int d, double N, const double F[3], double c, double out[4]) { flux_fn(d, N, F, c, out); }

/* HLL flux between a left state (Ul, flux gl) and a right state (Ur, gr) with signal speeds sm <= 0 <= sp */
void orc_hll_flux(const double Ul[4], const double gl[4], const double Ur[4], const double gr[4], double sm,
                  double sp, double out[4]) {
    for (int v = 0; v < 4; v++) {
        if (sp - sm > 0.0) out[v] = (sp * gl[v] - sm * gr[v] + sp * sm * (Ur[v] - Ul[v])) / (sp - sm);
        else out[v] = 0.5 * (gl[v] + gr[v]);       /* both states are beams across the face: nothing crosses it */
    }
}

static void hll_face(int d, const double Ul[4], const double Ur[4], double c, double out[4]) {
    double gl[4], gr[4], a, b, sm = 0.0, sp = 0.0;
    flux_fn(d, Ul[0], Ul + 1, c, gl);
    flux_fn(d, Ur[0], Ur + 1, c, gr);
    orc_m1_wavespeeds(Ul[0], Ul + 1, c, d, &a, &b);
    if (a < sm) sm = a;
    if (b > sp) sp = b;
    orc_m1_wavespeeds(Ur[0], Ur + 1, c, d, &a, &b);
    if (a < sm) sm = a;
    if (b > sp) sp = b;
    orc_hll_flux(Ul, gl, Ur, gr, sm, sp, out);
}

void orc_transport_hll(int nx, int ny, int nz, const double *N, const double *Fx, const double *Fy,
                       const double *Fz, double c, double dx, double dt,
                       double *N1, double *Fx1, double *Fy1, double *Fz1) {
    const long sx = 1, sy = nx, sz = (long)nx * ny;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                long id = i * sx + j * sy + k * sz;
                double U[4] = {N[id], Fx[id], Fy[id], Fz[id]};
                double Un[4] = {U[0], U[1], U[2], U[3]};
                for (int d = 0; d < 3; d++) {
                    long ip, im;
                    if (d == 0) { ip = wrap(i + 1, nx) * sx + j * sy + k * sz; im = wrap(i - 1, nx) * sx + j * sy + k * sz; }
                    else if (d == 1) { ip = i * sx + wrap(j + 1, ny) * sy + k * sz; im = i * sx + wrap(j - 1, ny) * sy + k * sz; }
                    else { ip = i * sx + j * sy + wrap(k + 1, nz) * sz; im = i * sx + j * sy + wrap(k - 1, nz) * sz; }
                    double Up[4] = {N[ip], Fx[ip], Fy[ip], Fz[ip]};
                    double Um[4] = {N[im], Fx[im], Fy[im], Fz[im]};
                    double f_hi[4], f_lo[4];
                    hll_face(d, U, Up, c, f_hi);                                 /* i+1/2 */
                    hll_face(d, Um, U, c, f_lo);                                 /* i-1/2 */
                    for (int v = 0; v < 4; v++) Un[v] -= dt / dx * (f_hi[v] - f_lo[v]);   /* Eq.A2 */
                }
                N1[id] = Un[0]; Fx1[id] = Un[1]; Fy1[id] = Un[2]; Fz1[id] = Un[3];
            }
}

/* ---------------------------------------------------------------------------------------------
 * O3 source injection.  S in Eq.3 / S_i^p in Eq.A2 (L66, L428); NGP, one emitter per cell (L103).
 * cell = floor(pos*n) mod n per axis (S11); N += rate*dt/dx^3; F unchanged (isotropic, S10).
 * ------------------------------------------------------------------------------------------- */
void orc_inject(int nx, int ny, int nz, double *N, long ns, const double *pos, const double *rate,
                double dt, double dx) {
    for (long s = 0; s < ns; s++) {
        long i = wrap((long)floor(pos[3 * s + 0] * nx), nx);
        long j = wrap((long)floor(pos[3 * s + 1] * ny), ny);
        long k = wrap((long)floor(pos[3 * s + 2] * nz), nz);
        N[i + (long)nx * (j + (long)ny * k)] += rate[s] * dt / (dx * dx * dx);
    }
}

/* ---------------------------------------------------------------------------------------------
 * Rate and cooling coefficients (reading S7; not printed in PAPER.md).
 * ------------------------------------------------------------------------------------------- */
void orc_rates(double T, orc_rates_t *r) {
    double lam = 2.0 * 157807.0 / T;
    double u, pw;
    /* recombination, Hui & Gnedin (1997) */
    r->alpha_A = 1.269e-13 * pow(lam, 1.503) / pow(1.0 + pow(lam / 0.522, 0.470), 1.923);
    r->alpha_B = 2.753e-14 * pow(lam, 1.500) / pow(1.0 + pow(lam / 2.740, 0.407), 2.242);
    /* collisional ionisation */
    u = pow(lam / 0.354, 0.874);
    r->beta = 21.11 * pow(T, -1.5) * exp(-0.5 * lam) * pow(lam, -1.089) / pow(1.0 + u, 1.101);
    r->z_ci = E0_EV * EV_ERG * r->beta;
    r->dl_ci = -1.5 + 0.5 * lam + 1.089 + 1.101 * 0.874 * u / (1.0 + u);
    /* recombination cooling, case A and B */
    u = pow(lam / 0.541, 0.502);
    r->z_recA = 1.778e-29 * T * pow(lam, 1.965) / pow(1.0 + u, 2.697);
    r->dl_recA = 1.0 - (1.965 - 2.697 * 0.502 * u / (1.0 + u));
    u = pow(lam / 2.250, 0.376);
    r->z_recB = 3.435e-30 * T * pow(lam, 1.970) / pow(1.0 + u, 3.720);
    r->dl_recB = 1.0 - (1.970 - 3.720 * 0.376 * u / (1.0 + u));
    /* collisional excitation (Cen 1992) */
    pw = sqrt(T / 1.0e5);
    r->z_exc = 7.5e-19 * exp(-118348.0 / T) / (1.0 + pw);
    r->dl_exc = 118348.0 / T - 0.5 * pw / (1.0 + pw);
    /* bremsstrahlung with Gaunt factor */
    {
        double L = log10(T);
        double gau = 0.34 * exp(-(5.5 - L) * (5.5 - L) / 3.0);
        double gff = 1.1 + gau;
        r->z_ff = 1.42e-27 * gff * sqrt(T);
        r->dl_ff = 0.5 + gau * (2.0 * (5.5 - L) / 3.0) / log(10.0) / gff;
    }
}

/* recombination clumping factor C_R from the cell's n_H (reading S8; Eq.15) */
double orc_clumping(double nH, const orc_params *p) {
    double C = 1.0;
    if (p->clump_model == 1) C = p->clump_a + p->clump_b * (nH / p->nH_mean - 1.0);
    else if (p->clump_model == 2) C = p->clump_a * pow(nH, p->clump_b);
    return C > 1.0 ? C : 1.0;
}

/* photon-atom cross clumping factor C_I of Eq.15 (L247-249): multiplies the photo-ionisation rate and,
 * so that every absorbed photon still ionises one atom, the absorption of N and F (reading S8b). */
double orc_clumping_i(double nH, const orc_params *p) {
    double C = 1.0;
    if (p->clump_i_a > 0.0) C = p->clump_i_a * pow(nH, p->clump_i_b);
    return C > 1.0 ? C : 1.0;
}

/* cooling function Lambda [erg cm^-3 s^-1] and its d/dlnT, at ionised fraction x, temperature T */
static void cooling_fn(double x, double T, double nH, double CR, const orc_rates_t *r,
                       const orc_params *p, double *Lam, double *Lam_T) {
    double y = 1.0 - x;
    double zrec = p->recomb_case == 1 ? r->z_recB : r->z_recA;
    double dlrec = p->recomb_case == 1 ? r->dl_recB : r->dl_recA;
    double zci = p->coll_ion ? r->z_ci : 0.0;
    *Lam = nH * nH * (x * x * (CR * zrec + r->z_ff) + x * y * (r->z_exc + zci));
    *Lam_T = nH * nH * (x * x * (CR * zrec * dlrec + r->z_ff * r->dl_ff)
                        + x * y * (r->z_exc * r->dl_exc + zci * r->dl_ci));
    if (p->redshift >= 0.0) {
        double zp1 = 1.0 + p->redshift;
        double k = 5.65e-36 * zp1 * zp1 * zp1 * zp1 * (x * nH);
        *Lam += k * (T - T_CMB0 * zp1);
        *Lam_T += k * T;
    }
}

/* ---------------------------------------------------------------------------------------------
 * O4 one chemistry sub-step of length dts (steps 4-5 of the algorithm in DESIGN.md / SURVEY O4):
 * backward-Euler, photon-conserving coupled update of (N, x) with lagged n_e and T, then the
 * linearly-implicit energy update.  In/out: N, F[3], x, T.  Returns absorbed photons per cm^3.
 *   dN/dt = -c sigma_n C_I n_H (1-x) N + S_rec                     (kappa terms of Eq.3-4)
 *   dx/dt = (1-x)(c sigma_n C_I N + beta n_e) - alpha C_R n_e x    (Eq.14-15, readings G2, S8b)
 * ------------------------------------------------------------------------------------------- */
double orc_chem_substep(double *N, double F[3], double *x_io, double *T_io, double nH, double dts,
                        const orc_params *p) {
    double x = *x_io, T = *T_io, y = 1.0 - x;
    orc_rates_t r;
    orc_rates(T, &r);
    double CR = orc_clumping(nH, p);
    double alpha = p->recomb_case == 1 ? r.alpha_B : r.alpha_A;
    double beta = p->coll_ion ? r.beta : 0.0;
    double ne = x * nH;
    double S_rec = p->recomb_case == 1 ? 0.0 : (r.alpha_A - r.alpha_B) * CR * ne * x * nH;
    double E = 1.5 * K_BOLTZ * nH * (1.0 + x) * T;

    double A = p->c * p->sigma_n * orc_clumping_i(nH, p) * nH * dts;
    double b = dts * beta * ne;
    double rr = dts * alpha * CR * ne;
    double L = 1.0 + b + rr;
    double Pq = (*N + dts * S_rec) / nH;
    double R0 = rr * x - b * y;
    double a2 = L * A;
    double a1 = L * (1.0 + A * y) + A * (Pq - R0);
    double a0 = Pq * A * y - R0 * (1.0 + A * y);
    double disc = sqrt(a1 * a1 - 4.0 * a2 * a0);
    double delta = (a1 >= 0.0) ? 2.0 * a0 / (a1 + disc) : (a1 - disc) / (2.0 * a2);
    double xn = x + delta;
    if (xn < 0.0) xn = 0.0;
    if (xn > 1.0) xn = 1.0;
    double yn = y - delta;
    double att = 1.0 / (1.0 + A * yn);
    double Nn = nH * Pq * att;
    double absorbed = A * yn * Nn;
    *N = Nn;
    F[0] *= att; F[1] *= att; F[2] *= att;          /* backward Euler of -kappa F (Eq.4) */
    *x_io = xn;
    if (p->cooling) {
        double e_erg = p->e_photon_eV * EV_ERG, e0 = E0_EV * EV_ERG;
        double dE_heat = absorbed * (e_erg * p->sigma_e / p->sigma_n - e0);
        double Lam, Lam_T;
        cooling_fn(xn, T, nH, CR, &r, p, &Lam, &Lam_T);
        double En = E + (dE_heat - dts * Lam) / (1.0 + dts * (Lam_T > 0.0 ? Lam_T : 0.0) / E);
        double Tn = En / (1.5 * K_BOLTZ * nH * (1.0 + xn));
        *T_io = Tn > T_MIN ? Tn : T_MIN;
    }
    return absorbed;
}

/* estimated net heating rate used to pick the sub-step (steps 2-3) */
static double edot_est(double N, double x, double T, double nH, const orc_params *p) {
    orc_rates_t r;
    orc_rates(T, &r);
    double CR = orc_clumping(nH, p);
    double e_erg = p->e_photon_eV * EV_ERG, e0 = E0_EV * EV_ERG;
    double H = nH * (1.0 - x) * p->c * orc_clumping_i(nH, p) * N * (e_erg * p->sigma_e - e0 * p->sigma_n);
    double Lam, Lam_T;
    cooling_fn(x, T, nH, CR, &r, p, &Lam, &Lam_T);
    return H - Lam;
}

/* O4 full per-cell operator Phi of Eq.A4 (L435-437): sub-cycled over the transport step dt.
 * `trace` (may be NULL) receives, for the first `trace_cap` sub-steps, the 4 numbers (dts, N, x, T) at the START of
 * each sub-step: the pin of the 10 % rule reads them; nothing is computed from them. */
int orc_chem_cell_trace(double *N, double F[3], double *x, double *T, double nH, double dt,
                        const orc_params *p, double *trace, int trace_cap) {
    double t_left = dt;
    int nsub = 0;
    while (t_left > 0.0 && nsub < p->max_sub) {
        double dts = t_left;
        if (p->cooling) {
            double E = 1.5 * K_BOLTZ * nH * (1.0 + *x) * (*T);
            double Ed = fabs(edot_est(*N, *x, *T, nH, p));
            if (Ed * t_left > p->eps_sub * E) dts = p->eps_sub * E / Ed;
        }
        if (trace && nsub < trace_cap) {
            trace[4 * nsub + 0] = dts; trace[4 * nsub + 1] = *N; trace[4 * nsub + 2] = *x; trace[4 * nsub + 3] = *T;
        }
        orc_chem_substep(N, F, x, T, nH, dts, p);
        t_left -= dts;
        nsub++;
    }
    return nsub;
}

int orc_chem_cell(double *N, double F[3], double *x, double *T, double nH, double dt,
                  const orc_params *p) {
    return orc_chem_cell_trace(N, F, x, T, nH, dt, p, NULL, 0);
}

/* Read-only views for the pins: out[0] = Lambda, out[1] = dLambda/dlnT of cooling_fn, out[2] = the net heating rate
 * H - Lambda that picks the sub-step (edot_est), all at (N, x, T, nH). */
void orc_cooling_probe(double N, double x, double T, double nH, const orc_params *p, double out[3]) {
    orc_rates_t r;
    orc_rates(T, &r);
    cooling_fn(x, T, nH, orc_clumping(nH, p), &r, p, &out[0], &out[1]);
    out[2] = edot_est(N, x, T, nH, p);
}

/* chemistry over the whole grid; returns total sub-cycles, *sub_max = largest per-cell count */
long long orc_chemistry(long ncell, double *N, double *Fx, double *Fy, double *Fz, double *x,
                        double *T, const double *nH, double dt, const orc_params *p,
                        long long *sub_max) {
    long long tot = 0, mx = 0;
#pragma omp parallel for schedule(dynamic, 4096) reduction(+ : tot) reduction(max : mx)
    for (long id = 0; id < ncell; id++) {
        double F[3] = {Fx[id], Fy[id], Fz[id]};
        int ns = orc_chem_cell(&N[id], F, &x[id], &T[id], nH[id], dt, p);
        Fx[id] = F[0]; Fy[id] = F[1]; Fz[id] = F[2];
        tot += ns;
        if (ns > mx) mx = ns;
    }
    *sub_max = mx;
    return tot;
}

/* ---------------------------------------------------------------------------------------------
 * O6 time loop: transport -> inject -> chemistry/cooling, n_steps times (order: PAPER.md:L411).
 * Fields are updated in place; stats[0] += total sub-cycles, stats[1] = max sub-cycles seen.
 * Returns 0, or -1 if scratch memory cannot be allocated.
 * ------------------------------------------------------------------------------------------- */
int orc_step(int nx, int ny, int nz, double *N, double *Fx, double *Fy, double *Fz, double *x,
             double *T, const double *nH, long ns, const double *pos, const double *rate,
             double dt, int n_steps, const orc_params *p, long long stats[2]) {
    long ncell = (long)nx * ny * nz;
    double *buf = (double *)malloc(sizeof(double) * 4 * ncell);
    if (!buf) return -1;
    double *N1 = buf, *Fx1 = buf + ncell, *Fy1 = buf + 2 * ncell, *Fz1 = buf + 3 * ncell;
    for (int s = 0; s < n_steps; s++) {
        if (p->flux == 1) orc_transport_hll(nx, ny, nz, N, Fx, Fy, Fz, p->c, p->dx, dt, N1, Fx1, Fy1, Fz1);
        else orc_transport(nx, ny, nz, N, Fx, Fy, Fz, p->c, p->dx, dt, N1, Fx1, Fy1, Fz1);
        memcpy(N, N1, sizeof(double) * ncell);
        memcpy(Fx, Fx1, sizeof(double) * ncell);
        memcpy(Fy, Fy1, sizeof(double) * ncell);
        memcpy(Fz, Fz1, sizeof(double) * ncell);
        orc_inject(nx, ny, nz, N, ns, pos, rate, dt, p->dx);
        long long mx = 0;
        stats[0] += orc_chemistry(ncell, N, Fx, Fy, Fz, x, T, nH, dt, p, &mx);
        if (mx > stats[1]) stats[1] = mx;
    }
    free(buf);
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * O5 global diagnostics (PAPER.md:L149 x_v, L303-305 mass-weighted, Eq.15 L249 Gamma = c sigma N).
 * out[0] <x>_V  [1] <x>_M  [2] <Gamma>_V  [3] <Gamma>_M  [4] photons_total = sum N dx^3
 * out[5] <T>_V  [6] max f = |F|/(cN) over cells with N>0  [7] min N  [8] # non-finite values
 * out[9] fraction of cells with x >= 0.5
 * ------------------------------------------------------------------------------------------- */
void orc_reduce(long ncell, const double *N, const double *Fx, const double *Fy, const double *Fz,
                const double *x, const double *T, const double *nH, const orc_params *p,
                double out[10]) {
    double sx = 0, sxm = 0, sm = 0, sg = 0, sgm = 0, sN = 0, sT = 0, fmax = 0, nmin = INFINITY;
    double nbad = 0, nhalf = 0;
    for (long id = 0; id < ncell; id++) {
        double gam = p->c * p->sigma_n * N[id];
        sx += x[id]; sxm += nH[id] * x[id]; sm += nH[id];
        sg += gam; sgm += nH[id] * gam; sN += N[id]; sT += T[id];
        if (N[id] > 0.0) {
            double f = sqrt(Fx[id] * Fx[id] + Fy[id] * Fy[id] + Fz[id] * Fz[id]) / (p->c * N[id]);
            if (f > fmax) fmax = f;
        }
        if (N[id] < nmin) nmin = N[id];
        if (!isfinite(N[id]) || !isfinite(Fx[id]) || !isfinite(Fy[id]) || !isfinite(Fz[id]) ||
            !isfinite(x[id]) || !isfinite(T[id])) nbad += 1;
        if (x[id] >= 0.5) nhalf += 1;
    }
    out[0] = sx / ncell; out[1] = sxm / sm; out[2] = sg / ncell; out[3] = sgm / sm;
    out[4] = sN * p->dx * p->dx * p->dx; out[5] = sT / ncell; out[6] = fmax; out[7] = nmin;
    out[8] = nbad; out[9] = nhalf / ncell;
}

/* =============================================================================================
 * Analysis and source front end around the step.  Not per step.
 * ============================================================================================= */

/* ---------------------------------------------------------------------------------------------
 * Clumping-factor measurement (section 3.2.1): "Clumping factors are computed by averaging the
 * relevant quantities on these 512 cells" of every b x b x b block (b = 8 in the paper: one cell of the coarse run),
 *     C_R = <n_H^2 x^2> / <n_H x>^2,          C_I = <n_gamma (1-x) n_H> / ( <n_gamma> <(1-x) n_H> )      (L247),
 * together with the block's mean density <n_H> and its ionised fraction <n_H x>/<n_H> (what the coarse cell holds;
 * the paper bins C_R, C_I against these two, Fig.12-13).  Where a denominator vanishes (no ionised gas / no photons /
 * no neutral gas) the factor is 1 (reading S21: a homogeneous block).  Outputs: [nz/b][ny/b][nx/b].
 * ------------------------------------------------------------------------------------------- */
void orc_clumping_blocks(int nx, int ny, int nz, int b, const double *nH, const double *x, const double *N,
                         double *out_nH, double *out_x, double *out_CR, double *out_CI) {
    int bx = nx / b, by = ny / b, bz = nz / b;
    double inv = 1.0 / ((double)b * b * b);
    for (int K = 0; K < bz; K++)
        for (int J = 0; J < by; J++)
            for (int I = 0; I < bx; I++) {
                double s_n = 0, s_nx = 0, s_n2x2 = 0, s_g = 0, s_yn = 0, s_gyn = 0;
                for (int k = K * b; k < (K + 1) * b; k++)
                    for (int j = J * b; j < (J + 1) * b; j++)
                        for (int i = I * b; i < (I + 1) * b; i++) {
                            long id = i + (long)nx * (j + (long)ny * k);
                            double n = nH[id], xx = x[id], g = N[id], yn = (1.0 - xx) * n;
                            s_n += n; s_nx += n * xx; s_n2x2 += n * n * xx * xx;
                            s_g += g; s_yn += yn; s_gyn += g * yn;
                        }
                long o = I + (long)bx * (J + (long)by * K);
                double m_n = s_n * inv, m_nx = s_nx * inv, m_g = s_g * inv, m_yn = s_yn * inv;
                out_nH[o] = m_n;
                out_x[o] = m_n > 0.0 ? m_nx / m_n : 0.0;
                out_CR[o] = m_nx > 0.0 ? (s_n2x2 * inv) / (m_nx * m_nx) : 1.0;
                out_CI[o] = (m_g > 0.0 && m_yn > 0.0) ? (s_gyn * inv) / (m_g * m_yn) : 1.0;
            }
}

/* ---------------------------------------------------------------------------------------------
 * 2-D distribution of two per-cell quantities (the J21(n_H), x(n_H), (1-x)(n_H) planes of PAPER.md Fig.5-19; L417
 * names histogramming as a GPU pattern).  Bin of a value v on an axis: floor((f(v) - lo)/(hi - lo) * nbins) with
 * f = log10 when `logscale`, v otherwise; values outside [lo, hi) (or <= 0 on a log axis) are not counted but
 * tallied in *outside.  counts[ib * na + ia].
 * ------------------------------------------------------------------------------------------- */
void orc_hist2d(long n, const double *a, const double *b, int log_a, int log_b, double a_lo, double a_hi,
                double b_lo, double b_hi, int na, int nb, long long *counts, long long *outside) {
    for (long k = 0; k < (long)na * nb; k++) counts[k] = 0;
    long long out = 0;
    for (long i = 0; i < n; i++) {
        double va = a[i], vb = b[i];
        if ((log_a && !(va > 0.0)) || (log_b && !(vb > 0.0))) { out++; continue; }
        double fa = log_a ? log10(va) : va, fb = log_b ? log10(vb) : vb;
        double ua = (fa - a_lo) / (a_hi - a_lo) * na, ub = (fb - b_lo) / (b_hi - b_lo) * nb;
        if (!(ua >= 0.0 && ua < (double)na && ub >= 0.0 && ub < (double)nb)) { out++; continue; }
        counts[(long)floor(ub) * na + (long)floor(ua)]++;
    }
    *outside = out;
}

/* ---------------------------------------------------------------------------------------------
 * Source front end (section 2.3, Eq.8-9).  For the transfer from t_p to t_{p+1} only the star
 * particles of snapshot p+1 are used.  With a_{p+1} the particle's age at t_{p+1}, a_p = a_{p+1} - (t_{p+1} - t_p),
 * L its lifetime as an ionising source and Ndot its intrinsic rate (photons_per_baryon * n_baryons / L):
 *   a_p > L                discarded;
 *   a_p < 0                born in the interval: "diluted" rate  (a_{p+1} / (t_{p+1} - t_p)) Ndot   -- the printed
 *                          "(a_{p+1} a*)/(t_{p+1} t_p)" lost its minus signs (reading G5): the star shone from its
 *                          birth a* to t_{p+1}, i.e. for a_{p+1} (at most L), spread over the interval;
 *   0 <= a_p <= L          min(1, (L - a_p)/(t_{p+1} - t_p)) Ndot  (it may stop shining inside the interval).
 * Every branch emits, over the interval, exactly the photons the star emits in it.  Then Eq.8: Ndot_eff = Ndot f_esc B
 * with the boost of Eq.9, read as B = max(1, a_b exp(k_b / t)) (reading G6: it is SFR_converged/SFR_actual >= 1 and
 * Table 1's a_b, k_b give B ~ 90 at 700 Myr for the 100 Mpc/h box; the printed "min" would switch it off), t = the age of
 * the Universe at the middle of the interval.
 * ------------------------------------------------------------------------------------------- */
double orc_boost(double t, double a_b, double k_b) {
    double B = a_b * exp(k_b / t);
    return B > 1.0 ? B : 1.0;
}

void orc_star_rates(long n, const double *age1, const double *life, const double *nbaryons, double photons_per_baryon,
                    double t_p, double t_p1, double f_esc, double a_b, double k_b, double *rate) {
    double dtp = t_p1 - t_p;
    double B = orc_boost(0.5 * (t_p + t_p1), a_b, k_b);
    for (long s = 0; s < n; s++) {
        double L = life[s], ndot = photons_per_baryon * nbaryons[s] / L;
        double a1 = age1[s], a0 = a1 - dtp, frac;
        if (a0 > L) frac = 0.0;
        else if (a0 < 0.0) frac = (a1 < L ? a1 : L) / dtp;
        else { frac = (L - a0) / dtp; if (frac > 1.0) frac = 1.0; }
        rate[s] = frac * ndot * f_esc * B;
    }
}

/* ---------------------------------------------------------------------------------------------
 * Thomson optical depth, Eq.10: tau = c sigma_T int n_e dt with n_e = x n_H, evaluated from a
 * history (z_i, x_i) of the mass-weighted ionised fraction in a flat LCDM background (the paper's WMAP-5 run, L45):
 *   n_H(z) = nH0 (1+z)^3,  dt = -dz / ((1+z) H(z)),  H = H0 sqrt(Om (1+z)^3 + 1 - Om)
 *   tau = c sigma_T nH0 int_0^zmax x(z) (1+z)^2 / H(z) dz   (trapezoid rule over the given points, z ascending).
 * ------------------------------------------------------------------------------------------- */
double orc_thomson_tau(long n, const double *z, const double *x, double nH0, double H0, double Om) {
    const double c = 2.99792458e10, sigma_T = 6.6524587e-25;
    double tau = 0.0;
    for (long i = 0; i + 1 < n; i++) {
        double f0 = x[i] * (1 + z[i]) * (1 + z[i]) / (H0 * sqrt(Om * pow(1 + z[i], 3) + 1.0 - Om));
        double f1 = x[i + 1] * (1 + z[i + 1]) * (1 + z[i + 1]) / (H0 * sqrt(Om * pow(1 + z[i + 1], 3) + 1.0 - Om));
        tau += 0.5 * (f0 + f1) * (z[i + 1] - z[i]);
    }
    return c * sigma_T * nH0 * tau;
}
