// Global diagnostics (O5): volume- and mass-weighted means of x and of the photo-ionisation rate
// (Eq.15), photon count, validity monitors.  Deterministic two-pass
// reduction: per-thread fp64 partials over 128-bit loads -> warp shuffles -> one row of partials per
// block -> a single block sums the rows in a fixed order.  (PAPER.md:L417 names reductions as the
// "naturally sequential" pattern that needs a specific technique on a GPU.)
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace aton {

enum { R_X = 0, R_XM, R_M, R_N, R_NM, R_T, R_F2MAX, R_NMIN, R_NHMIN, R_BAD, R_HALF, R_COUNT };

__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v) {
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_min(double v) {
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

__device__ __forceinline__ void block_combine(double acc[R_COUNT], double *out_row) {
    __shared__ double sh[32][R_COUNT];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
    for (int q = 0; q < R_COUNT; q++) {
        double v = (q == R_F2MAX) ? warp_max(acc[q]) : (q == R_NMIN || q == R_NHMIN) ? warp_min(acc[q]) : warp_sum(acc[q]);
        if (lane == 0) sh[w][q] = v;
    }
    __syncthreads();
    if (threadIdx.x < R_COUNT) {
        const int q = threadIdx.x;
        double v = sh[0][q];
        for (int i = 1; i < nw; i++)
            v = (q == R_F2MAX) ? fmax(v, sh[i][q]) : (q == R_NMIN || q == R_NHMIN) ? fmin(v, sh[i][q]) : v + sh[i][q];
        out_row[q] = v;
    }
}

// pass 1: each block writes partials[blockIdx.x][R_COUNT].  Any of N..T may be null (skipped, only
// n_H statistics are then produced -- used by aton_set_fields for <n_H> and the n_H > 0 check).
__global__ void __launch_bounds__(256) reduce_pass1(const float4 *__restrict__ N, const float4 *__restrict__ Gx,
                                                    const float4 *__restrict__ Gy, const float4 *__restrict__ Gz,
                                                    const float4 *__restrict__ x, const float4 *__restrict__ T,
                                                    const float4 *__restrict__ nH, int nquad, double *partials) {
    double acc[R_COUNT];
#pragma unroll
    for (int q = 0; q < R_COUNT; q++) acc[q] = 0.0;
    acc[R_NMIN] = INFINITY; acc[R_NHMIN] = INFINITY;
    const bool full = N != nullptr;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nquad; i += gridDim.x * blockDim.x) {
        const float4 h4 = __ldg(nH + i);
        const float h[4] = {h4.x, h4.y, h4.z, h4.w};
        float n[4] = {0, 0, 0, 0}, gx[4] = {0, 0, 0, 0}, gy[4] = {0, 0, 0, 0}, gz[4] = {0, 0, 0, 0}, xx[4] = {0, 0, 0, 0}, tt[4] = {0, 0, 0, 0};
        if (full) {
            float4 v;
            v = __ldg(N + i); n[0] = v.x; n[1] = v.y; n[2] = v.z; n[3] = v.w;
            v = __ldg(Gx + i); gx[0] = v.x; gx[1] = v.y; gx[2] = v.z; gx[3] = v.w;
            v = __ldg(Gy + i); gy[0] = v.x; gy[1] = v.y; gy[2] = v.z; gy[3] = v.w;
            v = __ldg(Gz + i); gz[0] = v.x; gz[1] = v.y; gz[2] = v.z; gz[3] = v.w;
            v = __ldg(x + i); xx[0] = v.x; xx[1] = v.y; xx[2] = v.z; xx[3] = v.w;
            v = __ldg(T + i); tt[0] = v.x; tt[1] = v.y; tt[2] = v.z; tt[3] = v.w;
        }
#pragma unroll
        for (int q = 0; q < 4; q++) {
            const double hd = h[q];
            acc[R_M] += hd;
            acc[R_NHMIN] = fmin(acc[R_NHMIN], hd);
            if (full) {
                acc[R_X] += xx[q];
                acc[R_XM] += hd * xx[q];
                acc[R_N] += n[q];
                acc[R_NM] += hd * n[q];
                acc[R_T] += tt[q];
                if (n[q] > 0.0f) {
                    const double rx = (double)gx[q] / n[q], ry = (double)gy[q] / n[q], rz = (double)gz[q] / n[q];
                    acc[R_F2MAX] = fmax(acc[R_F2MAX], rx * rx + ry * ry + rz * rz);
                }
                acc[R_NMIN] = fmin(acc[R_NMIN], (double)n[q]);
                const float chk = n[q] + gx[q] + gy[q] + gz[q] + xx[q] + tt[q];     // NaN/Inf poisons the sum
                if (!isfinite(n[q]) || !isfinite(gx[q]) || !isfinite(gy[q]) || !isfinite(gz[q]) ||
                    !isfinite(xx[q]) || !isfinite(tt[q]) || chk != chk) acc[R_BAD] += 1.0;
                if (xx[q] >= 0.5f) acc[R_HALF] += 1.0;
            }
        }
    }
    block_combine(acc, partials + (size_t)blockIdx.x * R_COUNT);
}

// pass 2: one block, fixed summation order over the rows
__global__ void __launch_bounds__(32) reduce_pass2(const double *partials, int nrows, double *out) {
    const int q = threadIdx.x;
    if (q >= R_COUNT) return;
    double v = partials[q];
    for (int r = 1; r < nrows; r++) {
        const double p = partials[(size_t)r * R_COUNT + q];
        v = (q == R_F2MAX) ? fmax(v, p) : (q == R_NMIN || q == R_NHMIN) ? fmin(v, p) : v + p;
    }
    out[q] = v;
}

__global__ void __launch_bounds__(256) scale_kernel(const float4 *__restrict__ in, float4 *out, float s, int nquad) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nquad; i += gridDim.x * blockDim.x) {
        float4 v = in[i];
        v.x *= s; v.y *= s; v.z *= s; v.w *= s;
        out[i] = v;
    }
}

// one bit per cell holding a source (variant 4's per-cell source flags); cells are unique
__global__ void __launch_bounds__(256) source_bits_kernel(const int *__restrict__ cells, int n, unsigned *bits) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) atomicOr(bits + ((unsigned)cells[s] >> 5), 1u << (cells[s] & 31));
}

}  // namespace aton
