// fp64 form of the sub-cycled chemistry / cooling operator Phi (Eq.13-15, Eq.A4; DESIGN.md
// reading S5) for the few cells where fp32 is not enough: near thermal balance the 10 % rule's sub-step
// eps E/|H - Lambda| divides by a difference that cancels, so the ~3e-6 of the fp32 rate fits decides which sub-step
// sequence is taken and the first-order sub-steps then differ at the per-cent level (H5).  The fp32
// loop (aton_physics.cuh, BAIL) detects the cancellation and hands the cell over; here every quantity of the
// sub-step -- rate fits, heating estimate, sub-step choice, quadratic, energy update -- is evaluated in double
// from the cell's fp32 inputs.  Same O(1) groups as the fp32 form (temperature units, A = c sigma n_H dt, P = N/n_H,
// unknown delta = x' - x); the fits are evaluated in natural-log space with libm-accurate exp / log.
#pragma once
#include "aton_physics.cuh"

namespace aton {

struct StepConstD {        // StepConst's constants in double (host-computed)
    double dt, cs, heat_K, heat_rate_K;
    double zrec0, zff0, zexc0, zci_over_beta, compton0, t_cmb, eps_sub;
    double clump_k0, clump_k1, ci_k0, ci_k1;
    int max_sub, clump_model;
};

struct RatesD {
    double alpha, d_alpha, beta;
    double zrec, zff, zxy, zrec_t, zff_t, zxy_t;
};

template <int FLAGS>
__device__ __noinline__ void rates_f64(double T, const StepConstD &c, RatesD &r) {
    constexpr bool CASE_A = FLAGS & F_CASE_A, COOL = FLAGS & F_COOL, COLL = FLAGS & F_COLL;
    const double invT = 1.0 / T, lam = 315614.0 * invT;                  // lambda = 2 * 157807 K / T
    const double LT = log(T), L = 12.662275226919286 - LT;               // ln lambda = ln 315614 - ln T
    // Hui & Gnedin (1997): alpha = K lam^p / (1 + (lam/l0)^q)^r
    const double uB = exp(0.407 * (L - 1.0079579203999789));                // ln 2.740
    const double aB = 2.753e-14 * exp(1.5 * L - 2.242 * log1p(uB));
    if (CASE_A) {
        const double uA = exp(0.470 * (L + 0.6500876910994983));             // -ln 0.522
        const double aA = 1.269e-13 * exp(1.503 * L - 1.923 * log1p(uA));
        r.alpha = aA;
        r.d_alpha = aA - aB;
    } else {
        r.alpha = aB;
        r.d_alpha = 0.0;
    }
    r.beta = 0.0;
    r.zrec = r.zff = r.zxy = r.zrec_t = r.zff_t = r.zxy_t = 0.0;
    double zci = 0.0, zci_t = 0.0;
    if (COLL) {
        const double u = exp(0.874 * (L + 1.0384583658483626));              // -ln 0.354
        const double l1u = log1p(u);
        // 21.11 T^-1.5 exp(-lam/2) lam^-1.089 / (1+u)^1.101
        r.beta = 21.11 * exp(-1.5 * LT - 0.5 * lam - 1.089 * L - 1.101 * l1u);
        if (COOL) {
            zci = r.beta * c.zci_over_beta;
            zci_t = zci * (-0.411 + 0.5 * lam + 0.962274 * (1.0 - exp(-l1u)));      // u/(1+u) = 1 - 1/(1+u)
        }
    }
    if (COOL) {
        // recombination cooling K T lam^p / (1+u)^r ; d ln/d ln T = 1 - p + r q u/(1+u)
        constexpr double q = CASE_A ? 0.502 : 0.376, ln_l0 = CASE_A ? -0.6143360001356556 : 0.8109302162163288;
        constexpr double p = CASE_A ? 1.965 : 1.970, rr = CASE_A ? 2.697 : 3.720;
        const double u = exp(q * (L - ln_l0)), iu = 1.0 / (1.0 + u);
        r.zrec = c.zrec0 * T * exp(p * L + rr * log(iu));
        r.zrec_t = r.zrec * (1.0 - p + rr * q * u * iu);
        // bremsstrahlung with Gaunt factor 1.1 + 0.34 exp(-(5.5 - log10 T)^2 / 3)
        const double d = 5.5 - LT * 0.4342944819032518;
        const double gau = 0.34 * exp(d * d * (-1.0 / 3.0)), gff = 1.1 + gau, sqT = sqrt(T);
        r.zff = c.zff0 * gff * sqT;
        r.zff_t = c.zff0 * sqT * (0.5 * gff + gau * d * 0.2895296546021679);          // (2/3)/ln 10
        // collisional excitation
        const double pw = sqT * 3.1622776601683794e-3, ipw = 1.0 / (1.0 + pw);          // sqrt(T / 1e5)
        const double zex = c.zexc0 * exp(-118348.0 * invT) * ipw;
        r.zxy = zex + zci;
        r.zxy_t = zex * (118348.0 * invT - 0.5 * pw * ipw) + zci_t;
    }
}

// In/out: N, G (after transport + injection), x, T; returns the sub-cycle count.
template <int FLAGS>
__device__ __noinline__ int chemistry_f64(double &N, double &gx, double &gy, double &gz, double &x, double &T, double nH,
                                          const StepConstD &c) {
    constexpr bool CASE_A = FLAGS & F_CASE_A, COOL = FLAGS & F_COOL;
    double CR = 1.0;
    if (c.clump_model == 1) CR = c.clump_k0 + c.clump_k1 * nH;
    else if (c.clump_model == 2) CR = c.clump_k0 * pow(nH, c.clump_k1);
    CR = fmax(CR, 1.0);
    const double CI = c.ci_k0 > 0.0 ? fmax(c.ci_k0 * pow(nH, c.ci_k1), 1.0) : 1.0;
    const double cs_nH = c.cs * nH * CI, heat_rate = c.heat_rate_K * CI, inv_nH = 1.0 / nH;
    double t_left = c.dt, att_tot = 1.0;
    int nsub = 0;
    while (t_left > 0.0 && nsub < c.max_sub) {
        RatesD r;
        rates_f64<FLAGS>(T, c, r);
        const double y = 1.0 - x, ne = x * nH, theta = (1.0 + x) * T;
        double dts = t_left;
        if (COOL) {
            const double lamK = nH * (x * x * (CR * r.zrec + r.zff) + x * y * r.zxy) + c.compton0 * x * (T - c.t_cmb);
            const double ed = fabs(y * N * heat_rate - lamK);
            if (ed * t_left > c.eps_sub * theta) dts = c.eps_sub * theta / ed;
        }
        const double A = cs_nH * dts, b = dts * r.beta * ne, rr = dts * r.alpha * CR * ne, L = 1.0 + b + rr;
        double P = N * inv_nH;
        if (CASE_A) P += dts * r.d_alpha * CR * ne * x;
        const double R0 = rr * x - b * y, onepAy = 1.0 + A * y;
        const double a2 = L * A, a1 = L * onepAy + A * (P - R0), a0 = P * A * y - R0 * onepAy;
        const double disc = sqrt(fmax(a1 * a1 - 4.0 * a2 * a0, 0.0));
        const double delta = a1 >= 0.0 ? 2.0 * a0 / (a1 + disc) : (a1 - disc) / (2.0 * a2);
        const double xn = fmin(fmax(x + delta, 0.0), 1.0), yn = fmax(y - delta, 0.0);
        const double att = 1.0 / (1.0 + A * yn), Pa = P * att;
        N = nH * Pa;
        att_tot *= att;
        if (COOL) {
            const double dth_heat = A * yn * Pa * c.heat_K;
            const double lamK = nH * (xn * xn * (CR * r.zrec + r.zff) + xn * yn * r.zxy) + c.compton0 * xn * (T - c.t_cmb);
            const double lamK_T = nH * (xn * xn * (CR * r.zrec_t + r.zff_t) + xn * yn * r.zxy_t) + c.compton0 * xn * T;
            const double thn = theta + (dth_heat - dts * lamK) * theta / (theta + dts * fmax(lamK_T, 0.0));
            T = fmax(thn / (1.0 + xn), 1.0);
        }
        x = xn;
        t_left -= dts;
        ++nsub;
    }
    gx *= att_tot; gy *= att_tot; gz *= att_tot;
    return nsub;
}

// One cell through Phi: the fp32 loop, redone in fp64 when it reports cancellation.  `inj` = photons / cm^3 injected by
// a source in this cell during the step (0 for almost every cell; fp64 so the stiff path sees the unrounded rate).
template <int FLAGS>
__device__ __forceinline__ int phi_cell(float &N, float &gx, float &gy, float &gz, float &x, float &T, float nH, double inj,
                                        const StepConst &c, const StepConstD &cd) {
    const float N0 = N, gx0 = gx, gy0 = gy, gz0 = gz, x0 = x, T0 = T;
    N += (float)inj;
    int ns = chemistry<FLAGS, true>(N, gx, gy, gz, x, T, nH, c);
    if (ns < 0) {
        double Nd = (double)N0 + inj, ax = gx0, ay = gy0, az = gz0, xd = x0, Td = T0;
        ns = chemistry_f64<FLAGS>(Nd, ax, ay, az, xd, Td, (double)nH, cd);
        N = (float)Nd; gx = (float)ax; gy = (float)ay; gz = (float)az; x = (float)xd; T = (float)Td;
    }
    return ns;
}

}  // namespace aton
