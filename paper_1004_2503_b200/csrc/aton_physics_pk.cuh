// Packed (two cells per thread-instruction) fp32 physics of the ATON step for the fused kernel
// (aton_step_fused.cuh): M1 closure (Eq.5-6) and ONE sub-step of the chemistry /
// cooling operator Phi (Eq.13-15, Eq.A4) taken over the whole transport
// step.  Same formulation as aton_physics.cuh (G = F/c, O(1) groups, solve for delta = x' - x, powers
// as ex2(p*lg2) on the MUFU unit); what differs is the execution shape:
//  * straight-line and branch-free: no sub-cycle loop.  The Anninos 10 % rule (reading S5)
//    is evaluated first; a cell that needs more than one sub-cycle is left untouched and flagged, and
//    the fix-up kernel runs the sub-cycled scalar operator (aton_physics.cuh) on it afterwards;
//  * every fp32 expression runs on an f2 pair (FFMA2/FADD2/FMUL2); MUFU, min/max and selects per half.
#pragma once
#include "aton_physics.cuh"
#include "aton_pk.cuh"

namespace aton {

// ---------------------------------------------------------------- O1 closure on a pair
// (a, s): P_dj = a*delta_dj + s*G_d*G_j.  N <= N_TINY: isotropic (a = N/3, s = 0), as in closure().
__device__ __forceinline__ void closure2(f2 N, f2 gx, f2 gy, f2 gz, f2 &a, f2 &s) {
    const float n0 = lo(N), n1 = hi(N);
    const f2 inv = pk(n0 > N_TINY ? m_rcp(n0) : 0.0f, n1 > N_TINY ? m_rcp(n1) : 0.0f);
    const f2 rx = gx * inv, ry = gy * inv, rz = gz * inv;
    const f2 ff = min2(fma2(rx, rx, fma2(ry, ry, rz * rz)), 1.0f);
    const f2 w = sqrt2(fma2(ff, -3.0f, 4.0f));
    a = (w - 1.0f) * (N * (1.0f / 3.0f));
    s = (inv * 3.0f) * rcp2(w + 2.0f);
}

// The same closure on ONE cell, operation for operation what closure2 does on each half (bit-identical): the x halo cell of
// a row segment is a single cell, and a scalar MUFU / FMUL costs half the pipe time of the packed form on a splat pair.
// Written with the _rn intrinsics so that every rounding is the one stated (none of closure2's operations is a bare
// product followed by an add, so nothing in it is contracted on either path).
__device__ __forceinline__ void closure1(float N, float gx, float gy, float gz, float &a, float &s) {
    const float inv = N > N_TINY ? m_rcp(N) : 0.0f;
    const float rx = __fmul_rn(gx, inv), ry = __fmul_rn(gy, inv), rz = __fmul_rn(gz, inv);
    const float ff = fminf(__fmaf_rn(rx, rx, __fmaf_rn(ry, ry, __fmul_rn(rz, rz))), 1.0f);
    const float w = m_sqrt(__fmaf_rn(ff, -3.0f, 4.0f));
    a = __fmul_rn(__fsub_rn(w, 1.0f), __fmul_rn(N, 1.0f / 3.0f));
    s = __fmul_rn(__fmul_rn(inv, 3.0f), m_rcp(__fadd_rn(w, 2.0f)));
}
// (U + sg F_x) of one cell, sg = +-1, with the roundings of the packed path as ptxas builds it: for the components
// whose flux is a bare product (F_Gy = t G_y, F_Gz = t G_z) it contracts mul.rn.f32x2 + add.rn.f32x2 of
// "u +- flux_row(0, ...)" into one FFMA2 (checked in SASS and bit for bit on 2^24 random cells), so U + sg t G is ONE
// fma here too; F_Gx = fma(t, G_x, a) is already an fma and is added with its own rounding.
__device__ __forceinline__ void xterm1(const float e[4], float a, float s, float sg, float w[4]) {
    const float t = __fmul_rn(s, e[1]);
    const float ts = __fmul_rn(t, sg);                       // exact
    w[0] = __fmaf_rn(e[1], sg, e[0]);
    w[1] = __fmaf_rn(__fmaf_rn(t, e[1], a), sg, e[1]);
    w[2] = __fmaf_rn(ts, e[2], e[2]);
    w[3] = __fmaf_rn(ts, e[3], e[3]);
}

// ---------------------------------------------------------------- rates on a pair (reading S7)
struct Rates2 {
    f2 alpha, d_alpha, beta;
    f2 zrec, zff, zxy;          // cooling coefficients / (1.5 kB)
    f2 zrec_t, zff_t, zxy_t;    // times d ln(zeta)/d ln T
};

template <int FLAGS>
__device__ __forceinline__ void rates2(f2 T, bool warm, const StepConst &c, Rates2 &r) {
    constexpr bool CASE_A = FLAGS & F_CASE_A, COOL = FLAGS & F_COOL, COLL = FLAGS & F_COLL;
    const f2 l2T = lg22(T);
    const f2 l2lam = 18.2678017f - l2T;                    // log2(2*157807/T)
    {   // Hui & Gnedin (1997): alpha = K lam^p / (1 + (lam/l0)^q)^r
        const f2 uB = ex22(fma2(l2lam, 0.407f, -0.407f * 1.45417589f));
        const f2 aB = ex22(fma2(l2lam, 1.5f, fma2(lg22(uB + 1.0f), -2.242f, -45.0459887f)));
        if (CASE_A) {
            const f2 uA = ex22(fma2(l2lam, 0.470f, 0.470f * 0.93787829f));
            const f2 aA = ex22(fma2(l2lam, 1.503f, fma2(lg22(uA + 1.0f), -1.923f, -42.8413732f)));
            r.alpha = aA;
            r.d_alpha = aA - aB;
        } else {
            r.alpha = aB;
            r.d_alpha = splat(0.0f);
        }
    }
    const f2 zero = splat(0.0f);
    r.beta = zero;
    r.zrec = r.zff = r.zxy = r.zrec_t = r.zff_t = r.zxy_t = zero;
    f2 sqT = zero;
    if (COOL) {
        // recombination cooling K T lam^p / (1+u)^r ; d ln/d ln T = 1 - p + r q u/(1+u)
        constexpr float q = CASE_A ? 0.502f : 0.376f, l0 = CASE_A ? 0.88629950f : -1.16992500f;
        constexpr float p = CASE_A ? 1.965f : 1.970f, rr = CASE_A ? 2.697f : 3.720f;
        const f2 u = ex22(fma2(l2lam, q, q * l0));
        const f2 lu = lg22(u + 1.0f);
        r.zrec = ex22((l2T + c.l2_zrec0) + fma2(l2lam, p, lu * -rr));
        r.zrec_t = r.zrec * fma2(u * (rr * q), rcp2(u + 1.0f), 1.0f - p);
        // bremsstrahlung with Gaunt factor: zff0 gff sqrt(T); zff_t = zff/2 + zff0 sqrt(T) gau d (2/3)/ln10
        sqT = sqrt2(T);
        const f2 d = fma2(l2T, -0.30102999f, 5.5f);                         // 5.5 - log10 T
        const f2 gau = ex22((d * d) * -0.48089835f) * 0.34f;               // 0.34 exp(-d^2/3)
        const f2 zs = sqT * c.zff0;
        r.zff = zs * (gau + 1.1f);
        r.zff_t = fma2(r.zff, 0.5f, (zs * gau) * (d * 0.28952965f));
    }
    // exp(-157807/T) and exp(-118348/T) underflow fp32 below 1100 K: `warm` (any cell of the thread above 1100 K) only
    // skips work, the skipped terms are exact zeros.  One branch holds all of it.
    if ((COLL || COOL) && warm) {
        const f2 invT = rcp2(T);
        f2 zci = zero, zci_t = zero;
        if (COLL) {
            const f2 lam = invT * 315614.0f;
            const f2 u = ex22(fma2(l2lam, 0.874f, 0.874f * 1.49817873f));      // (lam/0.354)^0.874
            const f2 lu = lg22(u + 1.0f);
            // log2 of T^-1.5 exp(-lam/2) lam^-1.089 / (1+u)^1.101
            const f2 e = fma2(l2T, -1.5f, fma2(lam, -0.72134752f, fma2(l2lam, -1.089f, lu * -1.101f)));
            r.beta = ex22(e + 4.39985467f);                                    // * 21.11
            if (COOL) {
                zci = r.beta * c.zci_over_beta;                                // 13.6 eV / (1.5 kB)
                zci_t = zci * (fma2(lam, 0.5f, -0.411f) + (u * 0.962274f) * rcp2(u + 1.0f));
            }
        }
        if (COOL) {     // collisional excitation
            const f2 pw = sqT * 3.16227766e-3f;                                 // sqrt(T/1e5)
            const f2 ipw = rcp2(pw + 1.0f);
            const f2 zex = (ex22(invT * -170740.07f) * c.zexc0) * ipw;         // 118348 * log2(e)
            const f2 zex_t = zex * fma2(invT, 118348.0f, (pw * ipw) * -0.5f);
            r.zxy = zex + zci;
            r.zxy_t = zex_t + zci_t;
        }
    }
}

__device__ __forceinline__ f2 clumping2(f2 nH, const StepConst &c) {
    if (c.clump_model == 1) return max2(fma2(nH, c.clump_k1, c.clump_k0), 1.0f);
    if (c.clump_model == 2) return max2(ex22(lg22(nH) * c.clump_k1) * c.clump_k0, 1.0f);
    return splat(1.0f);
}

// ---------------------------------------------------------------- O4, one sub-step of length dt
// In/out: N, G (after transport + injection), x, T.  Returns a 2-bit mask: bit h set = half h needs
// sub-cycling (its values are returned unchanged).  `force`: halves to leave unchanged and report
// whatever the 10 % rule says (variant 4 hands its source cells to the fix-up kernel this way).
template <int FLAGS>
__device__ __forceinline__ unsigned chem_fast2(f2 &N, f2 &gx, f2 &gy, f2 &gz, f2 &x, f2 &T, f2 nH,
                                               const StepConst &c, unsigned force = 0u) {
    constexpr bool CASE_A = FLAGS & F_CASE_A, COOL = FLAGS & F_COOL;
    const bool warm = fmaxf(lo(T), hi(T)) > 1100.0f;
    Rates2 r;
    rates2<FLAGS>(T, warm, c, r);
    const f2 CR = clumping2(nH, c);
    const bool ci_on = c.ci_k0 > 0.0f;                                    // uniform: C_I of Eq.15, off by default
    f2 nHs = nH, Ns = N;                                                  // C_I nH (absorbers seen by the photons), C_I N
    if (ci_on) {
        const f2 CI = max2(ex22(lg22(nH) * c.ci_k1) * c.ci_k0, 1.0f);
        nHs = nH * CI;
        Ns = N * CI;
    }
    const f2 y = 1.0f - x;
    const f2 ne = x * nH;
    const f2 theta = fma2(x, T, T);                                      // (1 + x) T
    const f2 crz = fma2(CR, r.zrec, r.zff);
    unsigned defer = force;
    if (COOL) {
        // estimated net heating rate / (1.5 kB nH) [K/s]: the Anninos 10 % rule decides on sub-cycling
        const f2 lamK = fma2(nH, (x * x) * crz + (x * y) * r.zxy, (x * c.compton0) * (T - c.t_cmb));
        const f2 ed = abs2(fma2(y * Ns, c.heat_rate_K, splat(0.0f) - lamK));
        const f2 lhs = ed * c.dt, rhs = theta * c.eps_sub;
        defer |= (lo(lhs) > lo(rhs) ? 1u : 0u) | (hi(lhs) > hi(rhs) ? 2u : 0u);
    }
    // backward-Euler coupled (N, x) update, solved for delta = x' - x
    const float dt = c.dt;
    const f2 A = (nHs * c.cs) * dt;
    const f2 dne = ne * dt;
    const f2 b = dne * r.beta;
    const f2 ane = (r.alpha * CR) * dne;                                  // rr = dt alpha C_R n_e
    const f2 L = (b + 1.0f) + ane;
    f2 P = N * rcp2(nH);
    if (CASE_A) P = fma2(((r.d_alpha * CR) * dne), x, P);                // + dt S_rec / nH
    const f2 R0 = ane * x - b * y;
    const f2 onepAy = fma2(A, y, 1.0f);
    const f2 a2 = L * A;
    const f2 a1 = fma2(L, onepAy, A * (P - R0));
    const f2 a0 = (P * A) * y - R0 * onepAy;
    const f2 disc = sqrt2(max2(fma2(a1, a1, (a2 * a0) * -4.0f), 0.0f));
    // delta = 2 a0/(a1 + disc) if a1 >= 0 else (a1 - disc)/(2 a2): pick numerator and denominator, one rcp
    const f2 den_p = a1 + disc, num_m = a1 - disc, num_p = a0 * 2.0f, den_m = a2 * 2.0f;
    const bool p0 = lo(a1) >= 0.0f, p1 = hi(a1) >= 0.0f;
    const f2 num = pk(p0 ? lo(num_p) : lo(num_m), p1 ? hi(num_p) : hi(num_m));
    const f2 den = pk(p0 ? lo(den_p) : lo(den_m), p1 ? hi(den_p) : hi(den_m));
    const f2 delta = num * rcp2(den);
    const f2 xn = min2(max2(x + delta, 0.0f), 1.0f);
    const f2 yn = max2(y - delta, 0.0f);
    const f2 att = rcp2(fma2(A, yn, 1.0f));
    const f2 Pa = P * att;
    f2 Tn = T;
    if (COOL) {
        const f2 dth_heat = ((A * yn) * Pa) * c.heat_K;
        const f2 xx = xn * xn, xy = xn * yn;
        const f2 ct = xn * c.compton0;
        const f2 lamK = fma2(nH, xx * crz + xy * r.zxy, ct * (T - c.t_cmb));
        const f2 lamK_T = fma2(nH, xx * fma2(CR, r.zrec_t, r.zff_t) + xy * r.zxy_t, ct * T);
        // theta' = theta + (dth_heat - dt lamK)/(1 + dt max(0, lamK_T)/theta)
        const f2 num_e = dth_heat - lamK * dt;
        const f2 thn = fma2(num_e * theta, rcp2(fma2(max2(lamK_T, 0.0f), dt, theta)), theta);
        Tn = max2(thn * rcp2(xn + 1.0f), 1.0f);
    }
    const f2 Nn = nH * Pa, gxn = gx * att, gyn = gy * att, gzn = gz * att;
    if (defer == 0u) {      // the common case by far: nothing to keep, no selects
        N = Nn; gx = gxn; gy = gyn; gz = gzn; x = xn; T = Tn;
    } else {                // a deferred half keeps its input values
        const bool k0 = defer & 1u, k1 = defer & 2u;
#define ATON_KEEP(old, nw) old = pk(k0 ? lo(old) : lo(nw), k1 ? hi(old) : hi(nw))
        ATON_KEEP(N, Nn); ATON_KEEP(gx, gxn); ATON_KEEP(gy, gyn); ATON_KEEP(gz, gzn);
        ATON_KEEP(x, xn); ATON_KEEP(T, Tn);
#undef ATON_KEEP
    }
    return defer;
}

}  // namespace aton
