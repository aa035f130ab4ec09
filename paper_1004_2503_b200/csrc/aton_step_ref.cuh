// Reference step kernel (variant 0): one thread per cell, the 7-point stencil gathered straight from
// global memory, closure recomputed for each neighbour, chemistry fused behind the transport update.
// It is the simplest statement of the fused step on the device: a cross-check for the product kernel
// (aton_step_v4.cuh), never the default.
#pragma once
#include "aton_physics_f64.cuh"

namespace aton {

struct Grid {
    int nx, ny, nz;
};

struct FieldsIO {
    const float *N, *Gx, *Gy, *Gz;      // step-p radiation fields (read only)
    float *N1, *Gx1, *Gy1, *Gz1;        // step-p+1 radiation fields (other buffer)
    float *x, *T;                       // updated in place (each cell reads only its own)
    const float *nH;
    const unsigned *src_mask;           // 1 bit per 32 consecutive cells: segment holds a source
    const int *src_cell;                // sorted flat cell indices of the sources
    const float *src_rho;               // rate / dx^3 per source cell [photons cm^-3 s^-1]
    const double *src_rho_d;            // the same, unrounded (the fp64 redo of stiff cells)
    int n_src;
    unsigned long long *stats;          // [0] += sub-cycles beyond one per cell, [1] = max sub-cycles, [2] += cells redone,
                                        // [3] += cells redone in fp64 (stiff)
    unsigned *defer_mask;               // variant 2: 1 bit per cell, set = needs sub-cycling (fix-up kernel clears it)
    const unsigned *src_bits;           // variant 4: 1 bit per cell, set = the cell holds a source
    int *stiff_q;                       // variant 4: [stiff_cap] ids of cells whose fp32 sub-cycling bailed out (they keep
    unsigned *stiff_n;                  //   their transported values); [0] = ids queued this step (may exceed the cap),
                                        //   [1] finished blocks of step_stiff_kernel, [2] group cursor and [3] finished
                                        //   blocks of step_fixup_kernel
    unsigned stiff_cap;
    int fix_inject;                     // 1: the redo paths inject the sources (variant 4); 0: the step kernel did (variant 2)
};

// index of flat cell `id` in the sorted source list, or -1 -- O3, NGP (L103)
__device__ __forceinline__ int source_find(const FieldsIO &f, int id) {
    int lo = 0, hi = f.n_src;
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (__ldg(f.src_cell + mid) < id) lo = mid + 1; else hi = mid;
    }
    return (lo < f.n_src && __ldg(f.src_cell + lo) == id) ? lo : -1;
}
// photons/cm^3 injected this step into flat cell `id` (0 for almost every cell)
__device__ __forceinline__ float source_lookup(const FieldsIO &f, int id, float dt) {
    const int s = source_find(f, id);
    return s >= 0 ? __ldg(f.src_rho + s) * dt : 0.0f;
}
__device__ __forceinline__ double source_lookup_d(const FieldsIO &f, int id, double dt) {
    const int s = source_find(f, id);
    return s >= 0 ? __ldg(f.src_rho_d + s) * dt : 0.0;
}

__device__ __forceinline__ bool source_segment_flag(const FieldsIO &f, int id) {
    if (f.n_src == 0) return false;
    unsigned seg = (unsigned)id >> 5;
    return (__ldg(f.src_mask + (seg >> 5)) >> (seg & 31)) & 1u;
}

// contribution of the neighbour at +e_d (sgn=+1) or -e_d (sgn=-1) to the LF update of the centre:
//   N  += h [ N_nb  - sgn * G_d,nb ]
//   G_j += h [ G_j,nb - sgn * P_dj,nb ],  P_dj = a delta_dj + s G_d G_j
template <int D>
__device__ __forceinline__ void add_neighbour(float sgn, float Nn, float gx, float gy, float gz,
                                              float &aN, float &ax, float &ay, float &az) {
    float a, s;
    closure(Nn, gx, gy, gz, a, s);
    const float gd = D == 0 ? gx : (D == 1 ? gy : gz);
    const float t = s * gd;
    float px = t * gx, py = t * gy, pz = t * gz;
    if (D == 0) px += a; else if (D == 1) py += a; else pz += a;
    aN += Nn - sgn * gd;
    ax += gx - sgn * px;
    ay += gy - sgn * py;
    az += gz - sgn * pz;
}

// ---------------------------------------------------------------------------------------------------
// HLL intercell flux (reading S20), in the units of the stored state
// U = (N, G = F/c), time in units of 1/c: flux rows FF_d = (G_d, P_dx, P_dy, P_dz), signal speeds in units of c.
//   FF_{i+1/2} = [ l+ FF_i - l- FF_{i+1} + l+ l- (U_{i+1} - U_i) ] / (l+ - l-),  l+ = max(0, hi_i, hi_{i+1}), l- = min(0, lo_i, lo_{i+1})
//   lo, hi = [ mu f -+ sqrt( (2/3)(xi^2 - xi) + 2 mu^2 (2 - f^2 - xi) ) ] / xi,   xi = sqrt(4 - 3 f^2), mu = G_d/|G|.
// fp32 form without the cancellations at f -> 0 and f -> 1: with r_d = mu f = G_d/N and g = 1 - f^2,
//   xi - 1 = 3 g/(xi + 1),  2 - f^2 - xi = -f^2 g/(2 - f^2 + xi)  =>  disc = g [ 2 xi/(xi + 1) - 2 r_d^2/(2 - f^2 + xi) ].
// ---------------------------------------------------------------------------------------------------
struct HllCell {
    float U[4];        // N, Gx, Gy, Gz
    float a, s;        // P_dj = a delta_dj + s G_d G_j
    float r[3];        // G_d / N, rescaled so that |r| <= 1 (f clamped, reading S2)
    float f2, xi;
};

__device__ __forceinline__ void hll_cell(float N, float gx, float gy, float gz, HllCell &c) {
    c.U[0] = N; c.U[1] = gx; c.U[2] = gy; c.U[3] = gz;
    closure(N, gx, gy, gz, c.a, c.s);
    float rx = 0.f, ry = 0.f, rz = 0.f, f2 = 0.f;
    if (N > N_TINY) {
        const float inv = f_rcp(N);
        rx = gx * inv; ry = gy * inv; rz = gz * inv;
        f2 = fmaf(rx, rx, fmaf(ry, ry, rz * rz));
        if (f2 > 1.0f) {
            const float sc = rsqrtf(f2);
            rx *= sc; ry *= sc; rz *= sc;
            f2 = 1.0f;
        }
    }
    c.r[0] = rx; c.r[1] = ry; c.r[2] = rz;
    c.f2 = f2;
    c.xi = f_sqrt(fmaf(-3.0f, f2, 4.0f));
}

template <int D>
__device__ __forceinline__ void hll_speeds(const HllCell &c, float &lo, float &hi) {
    const float g = 1.0f - c.f2, rd = c.r[D];
    const float disc = g * (2.0f * c.xi * f_rcp(c.xi + 1.0f) - 2.0f * rd * rd * f_rcp(2.0f - c.f2 + c.xi));
    const float root = f_sqrt(fmaxf(disc, 0.0f)), ixi = f_rcp(c.xi);
    lo = (rd - root) * ixi;
    hi = (rd + root) * ixi;
}

template <int D>
__device__ __forceinline__ void hll_flux_row(const HllCell &c, float F[4]) {
    const float gd = c.U[1 + D], t = c.s * gd;
    F[0] = gd;
    F[1] = t * c.U[1] + (D == 0 ? c.a : 0.0f);
    F[2] = t * c.U[2] + (D == 1 ? c.a : 0.0f);
    F[3] = t * c.U[3] + (D == 2 ? c.a : 0.0f);
}

// flux through the face between `l` (at -e_D) and `r` (at +e_D)
template <int D>
__device__ __forceinline__ void hll_face(const HllCell &l, const HllCell &r, float out[4]) {
    float Fl[4], Fr[4], lol, hil, lor, hir;
    hll_flux_row<D>(l, Fl);
    hll_flux_row<D>(r, Fr);
    hll_speeds<D>(l, lol, hil);
    hll_speeds<D>(r, lor, hir);
    const float sp = fmaxf(0.0f, fmaxf(hil, hir)), sm = fminf(0.0f, fminf(lol, lor));
    const float den = sp - sm;
    if (den > 0.0f) {
        const float inv = 1.0f / den, spm = sp * sm;
#pragma unroll
        for (int v = 0; v < 4; v++) out[v] = (sp * Fl[v] - sm * Fr[v] + spm * (r.U[v] - l.U[v])) * inv;
    } else {
#pragma unroll
        for (int v = 0; v < 4; v++) out[v] = 0.5f * (Fl[v] + Fr[v]);
    }
}

template <int D>
__device__ __forceinline__ void hll_axis(const HllCell &c, const FieldsIO &f, int idp, int idm, float mu, float Un[4]) {
    HllCell p, m;
    hll_cell(__ldg(f.N + idp), __ldg(f.Gx + idp), __ldg(f.Gy + idp), __ldg(f.Gz + idp), p);
    hll_cell(__ldg(f.N + idm), __ldg(f.Gx + idm), __ldg(f.Gy + idm), __ldg(f.Gz + idm), m);
    float fhi[4], flo[4];
    hll_face<D>(c, p, fhi);
    hll_face<D>(m, c, flo);
#pragma unroll
    for (int v = 0; v < 4; v++) Un[v] -= mu * (fhi[v] - flo[v]);
}

// one thread per cell: HLL transport, injection, chemistry (the structure of step_ref_kernel)
template <int FLAGS>
__global__ void __launch_bounds__(256) step_hll_kernel(FieldsIO f, Grid g, StepConst c, StepConstD cd) {
    const int ncell = g.nx * g.ny * g.nz;
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    int nsub = 0;
    if (id < ncell) {
        const int i = id % g.nx, j = (id / g.nx) % g.ny, k = id / (g.nx * g.ny);
        const int ip = (i + 1 == g.nx) ? 0 : i + 1, im = (i == 0) ? g.nx - 1 : i - 1;
        const int jp = (j + 1 == g.ny) ? 0 : j + 1, jm = (j == 0) ? g.ny - 1 : j - 1;
        const int kp = (k + 1 == g.nz) ? 0 : k + 1, km = (k == 0) ? g.nz - 1 : k - 1;
        const int row = g.nx * (j + g.ny * k);
        HllCell ce;
        hll_cell(__ldg(f.N + id), __ldg(f.Gx + id), __ldg(f.Gy + id), __ldg(f.Gz + id), ce);
        float Un[4] = {ce.U[0], ce.U[1], ce.U[2], ce.U[3]};
        const float mu = 2.0f * c.h;                       // c dt / dx
        hll_axis<0>(ce, f, ip + row, im + row, mu, Un);
        hll_axis<1>(ce, f, i + g.nx * (jp + g.ny * k), i + g.nx * (jm + g.ny * k), mu, Un);
        hll_axis<2>(ce, f, i + g.nx * (j + g.ny * kp), i + g.nx * (j + g.ny * km), mu, Un);
        float N = Un[0], gx = Un[1], gy = Un[2], gz = Un[3];
        const double inj = source_segment_flag(f, id) ? source_lookup_d(f, id, cd.dt) : 0.0;
        float x = f.x[id], T = f.T[id];
        nsub = phi_cell<FLAGS>(N, gx, gy, gz, x, T, __ldg(f.nH + id), inj, c, cd);
        f.N1[id] = N; f.Gx1[id] = gx; f.Gy1[id] = gy; f.Gz1[id] = gz;
        f.x[id] = x; f.T[id] = T;
    }
    int sum = nsub, mx = nsub;
    for (int o = 16; o > 0; o >>= 1) {
        sum += __shfl_xor_sync(0xffffffffu, sum, o);
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((threadIdx.x & 31) == 0 && sum > 0) {
        atomicAdd(f.stats, (unsigned long long)sum);
        atomicMax(f.stats + 1, (unsigned long long)mx);
    }
}

template <int FLAGS>
__global__ void __launch_bounds__(256) step_ref_kernel(FieldsIO f, Grid g, StepConst c, StepConstD cd) {
    const int ncell = g.nx * g.ny * g.nz;
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    int nsub = 0;
    if (id < ncell) {
        const int i = id % g.nx, j = (id / g.nx) % g.ny, k = id / (g.nx * g.ny);
        const int ip = (i + 1 == g.nx) ? 0 : i + 1, im = (i == 0) ? g.nx - 1 : i - 1;
        const int jp = (j + 1 == g.ny) ? 0 : j + 1, jm = (j == 0) ? g.ny - 1 : j - 1;
        const int kp = (k + 1 == g.nz) ? 0 : k + 1, km = (k == 0) ? g.nz - 1 : k - 1;
        const int row = g.nx * (j + g.ny * k);
        const int nb[6] = {ip + row, im + row, i + g.nx * (jp + g.ny * k), i + g.nx * (jm + g.ny * k),
                           i + g.nx * (j + g.ny * kp), i + g.nx * (j + g.ny * km)};
        float aN = 0.f, ax = 0.f, ay = 0.f, az = 0.f;
#define NB(D, SGN, Q) add_neighbour<D>(SGN, __ldg(f.N + nb[Q]), __ldg(f.Gx + nb[Q]), __ldg(f.Gy + nb[Q]), \
                                       __ldg(f.Gz + nb[Q]), aN, ax, ay, az)
        NB(0, 1.f, 0); NB(0, -1.f, 1); NB(1, 1.f, 2); NB(1, -1.f, 3); NB(2, 1.f, 4); NB(2, -1.f, 5);
#undef NB
        float N = fmaf(c.h, aN, c.keep * __ldg(f.N + id));
        float gx = fmaf(c.h, ax, c.keep * __ldg(f.Gx + id));
        float gy = fmaf(c.h, ay, c.keep * __ldg(f.Gy + id));
        float gz = fmaf(c.h, az, c.keep * __ldg(f.Gz + id));
        const double inj = source_segment_flag(f, id) ? source_lookup_d(f, id, cd.dt) : 0.0;
        float x = f.x[id], T = f.T[id];
        nsub = phi_cell<FLAGS>(N, gx, gy, gz, x, T, __ldg(f.nH + id), inj, c, cd);
        f.N1[id] = N; f.Gx1[id] = gx; f.Gy1[id] = gy; f.Gz1[id] = gz;
        f.x[id] = x; f.T[id] = T;
    }
    // sub-cycle statistics: block reduce, one atomic pair per block
    __shared__ int s_sum[8], s_max[8];
    int sum = nsub, mx = nsub;
    for (int o = 16; o > 0; o >>= 1) {
        sum += __shfl_xor_sync(0xffffffffu, sum, o);
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((threadIdx.x & 31) == 0) { s_sum[threadIdx.x >> 5] = sum; s_max[threadIdx.x >> 5] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int nw = (blockDim.x + 31) >> 5;
        for (int w = 1; w < nw; w++) { sum += s_sum[w]; mx = max(mx, s_max[w]); }
        atomicAdd(f.stats, (unsigned long long)sum);
        atomicMax(f.stats + 1, (unsigned long long)mx);
    }
}

}  // namespace aton
