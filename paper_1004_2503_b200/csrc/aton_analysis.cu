// Analysis and source front end around the step (none of it runs per step):
//  * aton_clumping_blocks  clumping factors C_R, C_I measured over b^3 blocks (section 3.2.1);
//  * aton_histogram2d      2-D distributions of two per-cell quantities, e.g. Gamma(n_H), x(n_H) (Fig.5-19;
//                          L417 names histogramming as a GPU pattern needing care);
//  * aton_set_star_sources star particles -> effective emission rates over a snapshot interval (section 2.3, Eq.8-9)
//                          -> aton_set_sources;
//  * aton_thomson_tau      Thomson optical depth of an ionisation history (Eq.10).
#include "aton_ctx.cuh"

namespace aton {

// ---------------------------------------------------------------------------------------------------------
// One warp per b^3 block: lanes stride over the block's cells in memory order (b consecutive x cells per row: 32-byte
// sectors for b = 8), fp32 loads, fp64 sums, shuffle reduction.  12 B per cell.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) clumping_blocks_kernel(const float *__restrict__ nH, const float *__restrict__ x,
                                                              const float *__restrict__ N, int nx, int ny, int b, int bx,
                                                              int by, long nblocks, float *o_nH, float *o_x, float *o_CR,
                                                              float *o_CI) {
    const int lane = threadIdx.x & 31;
    const long warp = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), nwarps = (long)gridDim.x * (blockDim.x >> 5);
    const int b2 = b * b, b3 = b2 * b;
    for (long o = warp; o < nblocks; o += nwarps) {
        const int I = (int)(o % bx), J = (int)((o / bx) % by), K = (int)(o / ((long)bx * by));
        double s_n = 0, s_nx = 0, s_n2x2 = 0, s_g = 0, s_yn = 0, s_gyn = 0;
        for (int c = lane; c < b3; c += 32) {
            const int i = c % b, j = (c / b) % b, k = c / b2;
            const long id = (long)(I * b + i) + (long)nx * ((J * b + j) + (long)ny * (K * b + k));
            const double n = __ldg(nH + id), xx = __ldg(x + id), g = __ldg(N + id), yn = (1.0 - xx) * n;
            s_n += n; s_nx += n * xx; s_n2x2 += n * n * xx * xx;
            s_g += g; s_yn += yn; s_gyn += g * yn;
        }
        for (int w = 16; w > 0; w >>= 1) {
            s_n += __shfl_xor_sync(0xffffffffu, s_n, w); s_nx += __shfl_xor_sync(0xffffffffu, s_nx, w);
            s_n2x2 += __shfl_xor_sync(0xffffffffu, s_n2x2, w); s_g += __shfl_xor_sync(0xffffffffu, s_g, w);
            s_yn += __shfl_xor_sync(0xffffffffu, s_yn, w); s_gyn += __shfl_xor_sync(0xffffffffu, s_gyn, w);
        }
        if (lane == 0) {
            const double inv = 1.0 / (double)b3;
            const double m_n = s_n * inv, m_nx = s_nx * inv, m_g = s_g * inv, m_yn = s_yn * inv;
            o_nH[o] = (float)m_n;
            o_x[o] = (float)(m_n > 0.0 ? m_nx / m_n : 0.0);
            o_CR[o] = (float)(m_nx > 0.0 ? (s_n2x2 * inv) / (m_nx * m_nx) : 1.0);          // reading S21
            o_CI[o] = (float)((m_g > 0.0 && m_yn > 0.0) ? (s_gyn * inv) / (m_g * m_yn) : 1.0);
        }
    }
}

// the per-cell quantities a histogram axis can show, evaluated in fp64 from the fp32 fields
__device__ __forceinline__ double quantity(int q, float nH, float x, float T, float N, double cs) {
    switch (q) {
        case ATON_Q_NH: return nH;
        case ATON_Q_X: return x;
        case ATON_Q_NEUTRAL: return 1.0 - (double)x;
        case ATON_Q_T: return T;
        case ATON_Q_N: return N;
        default: return cs * (double)N;      // ATON_Q_GAMMA = c sigma_n N (Eq.15)
    }
}

// Block-private histogram in shared memory (32-bit counts, at most 4096 bins), merged with 64-bit global atomics.
// The bin of a value is decided in fp64 exactly as the oracle does it.
__global__ void __launch_bounds__(256) hist2d_kernel(const float *__restrict__ nH, const float *__restrict__ x,
                                                     const float *__restrict__ T, const float *__restrict__ N, long ncell,
                                                     double cs, int qa, int qb, int log_a, int log_b, double a_lo,
                                                     double a_sc, double b_lo, double b_sc, int na, int nb,
                                                     unsigned long long *counts, unsigned long long *outside) {
    extern __shared__ unsigned hist[];
    const int nbins = na * nb;
    for (int k = threadIdx.x; k < nbins; k += blockDim.x) hist[k] = 0u;
    __syncthreads();
    unsigned out = 0;
    for (long id = (long)blockIdx.x * blockDim.x + threadIdx.x; id < ncell; id += (long)gridDim.x * blockDim.x) {
        const float h = __ldg(nH + id), xx = __ldg(x + id), t = __ldg(T + id), n = __ldg(N + id);
        const double va = quantity(qa, h, xx, t, n, cs), vb = quantity(qb, h, xx, t, n, cs);
        if ((log_a && !(va > 0.0)) || (log_b && !(vb > 0.0))) { out++; continue; }
        const double ua = ((log_a ? log10(va) : va) - a_lo) * a_sc, ub = ((log_b ? log10(vb) : vb) - b_lo) * b_sc;
        if (!(ua >= 0.0 && ua < (double)na && ub >= 0.0 && ub < (double)nb)) { out++; continue; }
        atomicAdd(&hist[(int)floor(ub) * na + (int)floor(ua)], 1u);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < nbins; k += blockDim.x)
        if (hist[k]) atomicAdd(counts + k, (unsigned long long)hist[k]);
    for (int w = 16; w > 0; w >>= 1) out += __shfl_xor_sync(0xffffffffu, out, w);
    if ((threadIdx.x & 31) == 0 && out) atomicAdd(outside, (unsigned long long)out);
}

// section 2.3: the three ageing branches, then f_esc * B (B formed once on the host: one scalar per interval)
__global__ void __launch_bounds__(256) star_rates_kernel(const double *__restrict__ age1, const double *__restrict__ life,
                                                         const double *__restrict__ nbar, long n, double ppb, double dtp,
                                                         double fesc_B, double *rate) {
    const long s = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const double L = life[s], ndot = ppb * nbar[s] / L, a1 = age1[s], a0 = a1 - dtp;
    double frac;
    if (a0 > L) frac = 0.0;
    else if (a0 < 0.0) frac = fmin(a1, L) / dtp;             // born inside the interval: diluted (reading G5)
    else frac = fmin((L - a0) / dtp, 1.0);                   // alive at its start; may stop shining inside it
    rate[s] = frac * ndot * fesc_B;
}

// Eq.10 by the trapezoid rule; one block, fixed summation order
__global__ void __launch_bounds__(256) thomson_tau_kernel(const double *__restrict__ z, const double *__restrict__ x, long n,
                                                          double H0, double Om, double pref, double *tau) {
    __shared__ double sh[256];
    double acc = 0.0;
    auto f = [&](long i) { const double q = 1.0 + z[i]; return x[i] * q * q / (H0 * sqrt(Om * q * q * q + 1.0 - Om)); };
    for (long i = threadIdx.x; i + 1 < n; i += blockDim.x) acc += 0.5 * (f(i) + f(i + 1)) * (z[i + 1] - z[i]);
    sh[threadIdx.x] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < 256; k++) t += sh[k];
        *tau = pref * t;
    }
}

}  // namespace aton

using namespace aton;

extern "C" {

int aton_clumping_blocks(aton_t *ctx, int block, float *nH_mean, float *x_mean, float *C_R, float *C_I, int on_device) {
    if (!ctx || !nH_mean || !x_mean || !C_R || !C_I) return ATON_EINVAL;
    if (!ctx->have_fields) return fail(ctx, ATON_ESTATE, "aton_clumping_blocks: no fields set");
    if (ctx->slab) return fail(ctx, ATON_ESTATE, "aton_clumping_blocks: undivided grids only");
    const Grid &g = ctx->g;
    if (block < 1 || g.nx % block || g.ny % block || g.nz % block)
        return fail(ctx, ATON_EINVAL, "aton_clumping_blocks: block %d must divide the grid %d x %d x %d", block, g.nx, g.ny, g.nz);
    cudaSetDevice(ctx->device);
    const int bx = g.nx / block, by = g.ny / block, bz = g.nz / block;
    const long nb = (long)bx * by * bz;
    float *out[4] = {nH_mean, x_mean, C_R, C_I}, *dev[4] = {nH_mean, x_mean, C_R, C_I};
    float *tmp = nullptr;
    if (!on_device) {
        CU(ctx, cudaMalloc((void **)&tmp, sizeof(float) * 4 * nb));
        for (int k = 0; k < 4; k++) dev[k] = tmp + k * nb;
    }
    const int blocks = (int)std::min<long>((nb + 7) / 8, 148L * 16);
    clumping_blocks_kernel<<<blocks, 256, 0, ctx->stream>>>(ctx->nH, ctx->x, ctx->rad[ctx->cur][0], g.nx, g.ny, block, bx, by,
                                                           nb, dev[0], dev[1], dev[2], dev[3]);
    ctx->launches++;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && !on_device)
        for (int k = 0; k < 4 && e == cudaSuccess; k++)
            e = cudaMemcpyAsync(out[k], dev[k], sizeof(float) * nb, cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(tmp);
    CU(ctx, e);
    return ATON_OK;
}

int aton_histogram2d(aton_t *ctx, int qa, int qb, int log_a, int log_b, double a_lo, double a_hi, double b_lo, double b_hi,
                     int na, int nb, long long *counts, long long *outside, int on_device) {
    if (!ctx || !counts || !outside) return ATON_EINVAL;
    if (!ctx->have_fields) return fail(ctx, ATON_ESTATE, "aton_histogram2d: no fields set");
    if (qa < 0 || qa > ATON_Q_GAMMA || qb < 0 || qb > ATON_Q_GAMMA) return fail(ctx, ATON_EINVAL, "aton_histogram2d: unknown quantity");
    if (na < 1 || nb < 1 || (long)na * nb > 4096 || !(a_hi > a_lo) || !(b_hi > b_lo))
        return fail(ctx, ATON_EINVAL, "aton_histogram2d: need 1 <= na * nb <= 4096 bins and hi > lo");
    cudaSetDevice(ctx->device);
    const int nbins = na * nb;
    unsigned long long *d = nullptr;
    unsigned long long *dc = (unsigned long long *)counts, *dout = (unsigned long long *)outside;
    if (!on_device) {
        CU(ctx, cudaMalloc((void **)&d, sizeof(unsigned long long) * (nbins + 1)));
        dc = d; dout = d + nbins;
    }
    cudaError_t e = cudaMemsetAsync(dc, 0, sizeof(unsigned long long) * nbins, ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(dout, 0, sizeof(unsigned long long), ctx->stream);
    if (e == cudaSuccess) {
        const size_t o = ctx->off;
        const long ncell = (long)ctx->ncell;
        const int blocks = (int)std::min<long>((ncell + 255) / 256, 148L * 8);
        hist2d_kernel<<<blocks, 256, sizeof(unsigned) * nbins, ctx->stream>>>(
            ctx->nH + o, ctx->x + o, ctx->T + o, ctx->rad[ctx->cur][0] + o, ncell, ctx->c * ctx->p.sigma_n, qa, qb, log_a, log_b,
            a_lo, (double)na / (a_hi - a_lo), b_lo, (double)nb / (b_hi - b_lo), na, nb, dc, dout);
        ctx->launches++;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess && !on_device) {
        e = cudaMemcpyAsync(counts, dc, sizeof(unsigned long long) * nbins, cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(outside, dout, sizeof(unsigned long long), cudaMemcpyDeviceToHost, ctx->stream);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(d);
    CU(ctx, e);
    return ATON_OK;
}

int aton_set_star_sources(aton_t *ctx, long long n, const float *pos, const double *age, const double *lifetime,
                          const double *nbaryons, double photons_per_baryon, double t_p, double t_p1, double f_esc,
                          double a_b, double k_b, int on_device) {
    if (!ctx) return ATON_EINVAL;
    if (n < 0 || (n > 0 && (!pos || !age || !lifetime || !nbaryons))) return fail(ctx, ATON_EINVAL, "aton_set_star_sources: bad arguments");
    if (!(t_p1 > t_p) || !(t_p > 0.0) || !(photons_per_baryon >= 0.0) || !(f_esc >= 0.0) || !(a_b >= 0.0))
        return fail(ctx, ATON_EINVAL, "aton_set_star_sources: need 0 < t_p < t_p1 and non-negative photons_per_baryon, f_esc, a_b");
    if (n == 0) return aton_set_sources(ctx, 0, nullptr, nullptr, 0);
    cudaSetDevice(ctx->device);
    // Eq.9 (reading G6): B = max(1, a_b exp(k_b / t)), t = the age of the Universe at the middle of the interval
    const double B = std::max(1.0, a_b * std::exp(k_b / (0.5 * (t_p + t_p1))));
    double *d = nullptr;
    float *dpos = nullptr;
    CU(ctx, cudaMalloc((void **)&d, sizeof(double) * 4 * n));
    cudaError_t e = cudaSuccess;
    const double *src[3] = {age, lifetime, nbaryons};
    const double *dv[3] = {age, lifetime, nbaryons};
    if (!on_device) {
        for (int k = 0; k < 3 && e == cudaSuccess; k++) {
            e = cudaMemcpyAsync(d + (k + 1) * n, src[k], sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream);
            dv[k] = d + (k + 1) * n;
        }
        if (e == cudaSuccess) e = cudaMalloc((void **)&dpos, sizeof(float) * 3 * n);
        if (e == cudaSuccess) e = cudaMemcpyAsync(dpos, pos, sizeof(float) * 3 * n, cudaMemcpyHostToDevice, ctx->stream);
    }
    int rc = ATON_OK;
    if (e == cudaSuccess) {
        star_rates_kernel<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(dv[0], dv[1], dv[2], (long)n, photons_per_baryon,
                                                                               t_p1 - t_p, f_esc * B, d);
        ctx->launches++;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) rc = aton_set_sources(ctx, n, on_device ? pos : dpos, d, 1);
    cudaFree(d);
    cudaFree(dpos);
    CU(ctx, e);
    return rc;
}

int aton_thomson_tau(aton_t *ctx, long long n, const double *z, const double *x, double nH0, double H0, double Om, double *tau) {
    if (!ctx || !z || !x || !tau || n < 2) return ATON_EINVAL;
    if (!(H0 > 0.0) || !(Om > 0.0) || !(Om <= 1.0) || !(nH0 >= 0.0)) return fail(ctx, ATON_EINVAL, "aton_thomson_tau: bad cosmology");
    for (long long i = 0; i + 1 < n; i++)
        if (!(z[i + 1] > z[i])) return fail(ctx, ATON_EINVAL, "aton_thomson_tau: z must ascend");
    cudaSetDevice(ctx->device);
    double *d = nullptr;
    CU(ctx, cudaMalloc((void **)&d, sizeof(double) * (2 * n + 1)));
    cudaError_t e = cudaMemcpyAsync(d, z, sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d + n, x, sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) {
        thomson_tau_kernel<<<1, 256, 0, ctx->stream>>>(d, d + n, (long)n, H0, Om, 2.99792458e10 * 6.6524587e-25 * nH0, d + 2 * n);
        ctx->launches++;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(tau, d + 2 * n, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(d);
    CU(ctx, e);
    return ATON_OK;
}

}  // extern "C"
