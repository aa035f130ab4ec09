// Per-cell fp32 physics of the ATON step for sm_100a: M1 closure (Eq.5-6) and the
// sub-cycled H photo-chemistry / cooling operator Phi (Eq.13-15, Eq.A4).
//
// Everything here is written for fp32 range and MUFU throughput:
//  * fluxes are carried as G = F/c, so the transport only contains mu = c dt/dx;
//  * the closure uses the division-free identity chi = (5 - 2w)/3, w = sqrt(4 - 3 f^2), which gives
//    P_dj = a delta_dj + s G_d G_j with a = (w-1) N/3 and s = 3/((2+w) N);
//  * chemistry works on O(1) groups (A = c sigma n_H dt, P = N/n_H, Theta = (1+x) T) with host
//    pre-scaled coefficients, and solves for delta = x' - x, never for 1 - x';
//  * powers are exp2(p*log2(.)) on the MUFU unit (ex2.approx / lg2.approx).
#pragma once
#include <cuda_runtime.h>

namespace aton {

// physics switches compiled into the kernels
enum : int { F_CASE_A = 1, F_COOL = 2, F_COLL = 4 };

struct StepConst {        // per aton_step call, host-computed in fp64, passed by value
    float h;              // mu/2 = c dt / (2 dx)
    float keep;           // 1 - 6h
    float dt;             // s
    float cs;             // c * sigma_n            [cm^3/s]
    float heat_K;         // (e sigma_e/sigma_n - e0)/(1.5 kB)   [K per absorbed photon per H atom]
    float heat_rate_K;    // c (e sigma_e - e0 sigma_n)/(1.5 kB) [K cm^3/s]
    float l2_zrec0;       // log2( zeta_rec prefactor / (1.5 kB) )  (case A or B)
    float zff0, zexc0;    // prefactors / (1.5 kB)
    float l2_zci0;        // log2( 13.6 eV * 21.11 / (1.5 kB) )
    float zci_over_beta;  // 13.6 eV / (1.5 kB)  [K]: zeta_ci = 13.6 eV * beta
    float compton0;       // 5.65e-36 (1+z)^4 / (1.5 kB), 0 when off
    float t_cmb;          // 2.726 (1+z)
    float eps_sub;
    int max_sub;
    int clump_model;
    float clump_k0, clump_k1;  // model 1: C = max(1, k0 + k1*nH); model 2: C = max(1, k0 * nH^k1)
    float ci_k0, ci_k1;   // C_I = max(1, k0 * nH^k1) on photo-ionisation and absorption; k0 <= 0: off (C_I = 1)
    float inj_scale;      // dt / dx^3 folded into the per-source density rate
    float stiff_kappa;    // BAIL: hand a cell to the fp64 path when |H - Lambda| < kappa (H + |Lambda|) limits a sub-step,
    float stiff_sens;     // ... when the attenuation's sensitivity to the sub-step partition, sum A y'/(1 + A y'), exceeds this
    int stiff_nsub;       // ... or when it needs more than this many sub-cycles
};

// ---------------------------------------------------------------- MUFU wrappers
__device__ __forceinline__ float f_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float f_sqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float f_ex2(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float f_lg2(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

constexpr float N_TINY = 1.0e-30f;   // below this N the closure is taken isotropic (fp32 range guard)

// ---------------------------------------------------------------- O1 closure
// (a, s) such that the pressure tensor is P_dj = a*delta_dj + s*G_d*G_j  (G = F/c).
__device__ __forceinline__ void closure(float N, float gx, float gy, float gz, float &a, float &s) {
    if (N > N_TINY) {
        float inv = f_rcp(N);
        float rx = gx * inv, ry = gy * inv, rz = gz * inv;
        float f2 = fminf(1.0f, fmaf(rx, rx, fmaf(ry, ry, rz * rz)));
        float w = f_sqrt(fmaf(-3.0f, f2, 4.0f));
        a = (w - 1.0f) * N * (1.0f / 3.0f);
        s = 3.0f * inv * f_rcp(2.0f + w);
    } else {
        a = N * (1.0f / 3.0f);
        s = 0.0f;
    }
}

// ---------------------------------------------------------------- rates (reading S7)
struct Rates {
    float alpha;      // recombination coefficient used in dx/dt (A or B)       [cm^3/s]
    float d_alpha;    // alpha_A - alpha_B (recombination radiation), case A only
    float beta;       // collisional ionisation                                  [cm^3/s]
    float zrec, zff, zxy;        // cooling coefficients / (1.5 kB): rec, ff, exc+ci  [K cm^3/s]
    float zrec_t, zff_t, zxy_t;  // the same times d ln(zeta)/d ln T
};

template <int FLAGS>
__device__ __forceinline__ void rates(float T, const StepConst &c, Rates &r) {
    constexpr bool CASE_A = FLAGS & F_CASE_A, COOL = FLAGS & F_COOL, COLL = FLAGS & F_COLL;
    const float l2T = f_lg2(T);
    const float invT = f_rcp(T);
    const float l2lam = 18.2678017f - l2T;                 // log2(2*157807) - log2 T
    const float lam = 315614.0f * invT;
    // Hui & Gnedin (1997): alpha = K lam^p / (1 + (lam/l0)^q)^r
    {
        float uB = f_ex2(0.407f * (l2lam - 1.45417589f));                       // (lam/2.740)^0.407
        float aB = f_ex2(fmaf(1.5f, l2lam, fmaf(-2.242f, f_lg2(1.0f + uB), -45.0459887f)));  // log2(2.753e-14)
        if (CASE_A) {
            float uA = f_ex2(0.470f * (l2lam + 0.93787829f));                   // (lam/0.522)^0.470
            float aA = f_ex2(fmaf(1.503f, l2lam, fmaf(-1.923f, f_lg2(1.0f + uA), -42.8413732f)));  // log2(1.269e-13)
            r.alpha = aA;
            r.d_alpha = aA - aB;
        } else {
            r.alpha = aB;
            r.d_alpha = 0.0f;
        }
    }
    r.beta = 0.0f;
    r.zrec = r.zff = r.zxy = r.zrec_t = r.zff_t = r.zxy_t = 0.0f;
    // Boltzmann factors exp(-157807/T), exp(-118348/T) are below the smallest fp32 denormal for
    // T < 1100 K: skipping them there is exact in fp32 (and they are 0 in the fp64 oracle < 200 K).
    const bool warm = T > 1100.0f;
    float zci = 0.0f, zci_t = 0.0f;
    if (COLL && warm) {
        float u = f_ex2(0.874f * (l2lam + 1.49817873f));                         // (lam/0.354)^0.874
        float lu = f_lg2(1.0f + u);
        // 21.11 T^-1.5 exp(-lam/2) lam^-1.089 / (1+u)^1.101
        float e = fmaf(-1.5f, l2T, fmaf(-0.72134752f, lam, fmaf(-1.089f, l2lam, -1.101f * lu)));
        r.beta = f_ex2(e + 4.39985467f);                                       // log2(21.11)
        if (COOL) {
            zci = f_ex2(e + c.l2_zci0);
            zci_t = zci * (fmaf(0.5f, lam, -0.411f) + 0.962274f * u * f_rcp(1.0f + u));
        }
    }
    if (COOL) {
        // recombination cooling: K T lam^p / (1+u)^r ; d ln/d ln T = 1 - p + r q u/(1+u)
        float u, lu, p, rq, rr;
        if (CASE_A) { u = f_ex2(0.502f * (l2lam + 0.88629950f)); p = 1.965f; rr = 2.697f; rq = 2.697f * 0.502f; }
        else        { u = f_ex2(0.376f * (l2lam - 1.16992500f)); p = 1.970f; rr = 3.720f; rq = 3.720f * 0.376f; }
        lu = f_lg2(1.0f + u);
        r.zrec = f_ex2(c.l2_zrec0 + l2T + fmaf(p, l2lam, -rr * lu));
        r.zrec_t = r.zrec * (1.0f - p + rq * u * f_rcp(1.0f + u));
        // bremsstrahlung with Gaunt factor
        float sqT = f_sqrt(T);
        float d = fmaf(-0.30102999f, l2T, 5.5f);                                     // 5.5 - log10 T
        float gau = 0.34f * f_ex2(-0.48089835f * d * d);                          // exp(-d^2/3)
        float gff = 1.1f + gau;
        r.zff = c.zff0 * gff * sqT;
        r.zff_t = r.zff * (0.5f + gau * d * 0.28952965f * f_rcp(gff));            // (2/3)/ln10
        // collisional excitation
        float zex = 0.0f, zex_t = 0.0f;
        if (warm) {
            float pw = sqT * 3.16227766e-3f;                                      // sqrt(T/1e5)
            float ipw = f_rcp(1.0f + pw);
            zex = c.zexc0 * f_ex2(-170740.07f * invT) * ipw;                      // 118348 * log2(e)
            zex_t = zex * fmaf(118348.0f, invT, -0.5f * pw * ipw);
        }
        r.zxy = zex + zci;
        r.zxy_t = zex_t + zci_t;
    }
}

__device__ __forceinline__ float clumping(float nH, const StepConst &c) {
    float C = 1.0f;
    if (c.clump_model == 1) C = fmaf(c.clump_k1, nH, c.clump_k0);
    else if (c.clump_model == 2) C = c.clump_k0 * f_ex2(c.clump_k1 * f_lg2(nH));
    return fmaxf(C, 1.0f);
}

// photon-atom cross clumping factor C_I of Eq.15
__device__ __forceinline__ float clumping_i(float nH, const StepConst &c) {
    return fmaxf(c.ci_k0 * f_ex2(c.ci_k1 * f_lg2(nH)), 1.0f);
}

// ---------------------------------------------------------------- O4 chemistry / cooling
// In/out: N, G (=F/c), x, T after transport + injection; nH fixed.  Returns the sub-cycle count.
// BAIL: give up (return -1, in/out values then meaningless) as soon as a sub-step is limited by the 10 % rule while
// heating and cooling cancel to better than STIFF_KAPPA: the sub-step eps E/|H - Lambda| is then ill-conditioned
// (the fp32 rate fits carry ~3e-6) and the caller redoes the cell with chemistry_f64 (aton_physics_f64.cuh).

// One cell on its way through the sub-cycled operator: chem_begin, then chem_substep until it returns non-zero.
struct ChemCell {
    float N, x, T, y;        // y = 1 - x is carried: y' = y - delta keeps the neutral fraction's own digits (H1)
    float nH, CR, inv_nH, cs_nH, heat_rate;
    float t_left, att_tot, sens;
    int nsub;
};

__device__ __forceinline__ void chem_begin(ChemCell &s, float N, float x, float T, float nH, const StepConst &c) {
    s.N = N; s.x = x; s.T = T; s.y = 1.0f - x;
    s.nH = nH;
    s.CR = clumping(nH, c);
    s.inv_nH = f_rcp(nH);
    const bool ci_on = c.ci_k0 > 0.0f;
    const float CI = ci_on ? clumping_i(nH, c) : 1.0f;
    s.cs_nH = ci_on ? c.cs * nH * CI : c.cs * nH;
    s.heat_rate = ci_on ? c.heat_rate_K * CI : c.heat_rate_K;
    s.t_left = c.dt;
    s.att_tot = 1.0f;
    s.sens = 0.0f;
    s.nsub = 0;
}

// One sub-step.  Returns 0: more to do; 1: the step is complete (s.N, s.x, s.T final, G *= s.att_tot); -1 (BAIL only): give up.
template <int FLAGS, bool BAIL>
__device__ __forceinline__ int chem_substep(ChemCell &s, const StepConst &c) {
    constexpr bool CASE_A = FLAGS & F_CASE_A, COOL = FLAGS & F_COOL;
    if (!(s.t_left > 0.0f) || s.nsub >= c.max_sub) return 1;
    if (BAIL && s.nsub >= c.stiff_nsub) return -1;
    const float N = s.N, x = s.x, T = s.T, y = s.y, nH = s.nH, CR = s.CR, t_left = s.t_left;
    Rates r;
    rates<FLAGS>(T, c, r);
    const float ne = x * nH;
    const float theta = (1.0f + x) * T;
    float dts = t_left;
    if (COOL) {
        // estimated net heating rate / (1.5 kB nH)  [K/s]
        float lamK = nH * (x * x * fmaf(CR, r.zrec, r.zff) + x * y * r.zxy) + c.compton0 * x * (T - c.t_cmb);
        const float heat = y * N * s.heat_rate;
        float ed = fabsf(heat - lamK);
        if (ed * t_left > c.eps_sub * theta) {
            if (BAIL && ed < c.stiff_kappa * (heat + fabsf(lamK))) return -1;
            dts = c.eps_sub * theta / ed;
        }
    }
    // backward-Euler coupled (N, x) update, solved for delta = x' - x
    const float A = s.cs_nH * dts;
    const float b = dts * r.beta * ne;
    const float rr = dts * r.alpha * CR * ne;
    const float L = 1.0f + b + rr;
    float P = N * s.inv_nH;
    if (CASE_A) P = fmaf(dts * r.d_alpha * CR * ne, x, P);       // + dts*S_rec/nH
    const float R0 = rr * x - b * y;
    const float onepAy = fmaf(A, y, 1.0f);
    const float a2 = L * A;
    const float a1 = fmaf(L, onepAy, A * (P - R0));
    const float a0 = fmaf(P * A, y, -R0 * onepAy);
    const float disc = f_sqrt(fmaxf(fmaf(a1, a1, -4.0f * a2 * a0), 0.0f));
    float delta;
    if (a1 >= 0.0f) delta = 2.0f * a0 * f_rcp(a1 + disc);
    else delta = (a1 - disc) * f_rcp(2.0f * a2);
    const float xn = fminf(fmaxf(x + delta, 0.0f), 1.0f);
    const float yn = fmaxf(y - delta, 0.0f);
    const float att = f_rcp(fmaf(A, yn, 1.0f));
    if (BAIL) {
        // How much the result moves per unit relative error of the sub-step lengths (the fp32 heating estimate that
        // sets them carries a few 1e-6).  Backward-Euler decay is partition sensitive wherever
        // rate x dts >> 1:  N' = prod_k (N + s_k)/(1 + A_k y'_k)  moves by  e g_N,  g_N = |s_k/(N + s_k) - A y'/(1 + A y')|
        // (s_k: the recombination photons of the sub-step), and a recombining x by  e g_x,  g_x = 1 - 1/L.  The LAST
        // sub-step takes what is left: it inherits minus the summed errors of the others, blown up by
        // dt/dts_last - 1 when it is a sliver.
        const float src = CASE_A ? 1.0f - N * s.inv_nH * f_rcp(P) : 0.0f;
        const float g = fmaxf(fabsf(src - (1.0f - att)), 1.0f - f_rcp(L));
        if (dts < t_left) {
            s.sens += g;
            if (s.sens > c.stiff_sens) return -1;
        } else if (s.nsub > 0 && s.sens + g * (c.dt * f_rcp(dts) - 1.0f) > c.stiff_sens) {
            return -1;
        }
    }
    const float Pa = P * att;
    s.N = nH * Pa;
    s.att_tot *= att;
    if (COOL) {
        const float dth_heat = A * yn * Pa * c.heat_K;
        const float lamK = nH * (xn * xn * fmaf(CR, r.zrec, r.zff) + xn * yn * r.zxy)
                           + c.compton0 * xn * (T - c.t_cmb);
        const float lamK_T = nH * (xn * xn * fmaf(CR, r.zrec_t, r.zff_t) + xn * yn * r.zxy_t)
                             + c.compton0 * xn * T;
        // theta' = theta + (dth_heat - dts lamK)/(1 + dts max(0,lamK_T)/theta)
        const float num = dth_heat - dts * lamK;
        const float thn = fmaf(num * theta, f_rcp(fmaf(dts, fmaxf(lamK_T, 0.0f), theta)), theta);
        s.T = fmaxf(thn * f_rcp(1.0f + xn), 1.0f);
    }
    s.x = xn;
    s.y = yn;
    s.t_left = t_left - dts;
    ++s.nsub;
    return (s.t_left > 0.0f && s.nsub < c.max_sub) ? 0 : 1;
}

template <int FLAGS, bool BAIL = false>
__device__ __forceinline__ int chemistry(float &N, float &gx, float &gy, float &gz, float &x, float &T,
                                         float nH, const StepConst &c) {
    ChemCell s;
    chem_begin(s, N, x, T, nH, c);
    int st;
    do st = chem_substep<FLAGS, BAIL>(s, c); while (st == 0);
    if (st < 0) return -1;
    N = s.N; x = s.x; T = s.T;
    gx *= s.att_tot; gy *= s.att_tot; gz *= s.att_tot;
    return s.nsub;
}

}  // namespace aton
