// aton_field_sums_noalloc (include/aton.h): the raw diagnostic sums of aton_reduce_sums (O5: PAPER.md:L149 volume-weighted x,
// L303-305 mass-weighted, Eq.15 L249 Gamma = c sigma_n N) for callers that must not allocate -- code under CUDA graph capture,
// serving loops, harnesses that forbid cudaMalloc.  No context, no cudaMalloc / cudaFree / allocating library call, no
// synchronisation: two kernel launches on the caller's stream, inputs and the output in the caller's device memory.
//
// It is a variant of the two-pass reduction of aton_reduce.cuh (reduce_pass1 / reduce_pass2) whose scratch -- one row of
// partial sums per block -- does not come from aton_init's cudaMalloc but from a file-scope static __device__ array below:
// NOALLOC_ROWS rows x 11 doubles = 104 192 bytes, held by every GPU that loads libaton.so until the process exits.
//  * every call on a device shares that array, and it keeps the last call's contents.  Nothing in it has to start at zero:
//    pass 1 writes rows [0, blocks) in full before pass 2 reads exactly those rows, so stale rows of a larger earlier call
//    are never read;
//  * two calls that OVERLAP on the GPU (different streams, or graphs replayed concurrently) race on the array.  Calls on one
//    stream are ordered and safe.
//  * in host code the array's name is a host-side stand-in, not a device address; the address is taken once per device with
//    cudaGetSymbolAddress (that device current) and passed to the kernels.
#include <cstdint>

#include "aton_ctx.cuh"

namespace {

enum { S_X = 0, S_XM, S_M, S_N, S_NM, S_T, S_F2MAX, S_NMIN, S_NHMIN, S_BAD, S_HALF, S_COUNT };   // = aton_reduce.cuh's rows
constexpr int NOALLOC_ROWS = 148 * 8;                 // blocks of pass 1 at most (the context path's REDUCE_BLOCKS)
constexpr long long NOALLOC_MAX_CELLS = 2147483644LL; // 2^31 - 4: 32-bit quad indices, as everywhere in the library
constexpr int MAX_DEVICES = 64;

static __device__ __align__(256) double g_noalloc_scratch[NOALLOC_ROWS * S_COUNT];

// device address of the array, per device (0 = not asked yet).  Host code must never hand g_noalloc_scratch itself to a kernel.
double *g_scratch_addr[MAX_DEVICES] = {};

__device__ __forceinline__ double wsum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double wmax(double v) {
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double wmin(double v) {
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ bool is_max_row(int q) { return q == S_F2MAX; }
__device__ __forceinline__ bool is_min_row(int q) { return q == S_NMIN || q == S_NHMIN; }

// pass 1: reduce_pass1's loop on F instead of G = F/c (the caller's arrays are the ABI's: photons cm^-2 s^-1);
// block b writes scratch row b
__global__ void __launch_bounds__(256) noalloc_pass1(const float4 *__restrict__ N, const float4 *__restrict__ Fx,
                                                     const float4 *__restrict__ Fy, const float4 *__restrict__ Fz,
                                                     const float4 *__restrict__ x, const float4 *__restrict__ T,
                                                     const float4 *__restrict__ nH, int nquad, double inv_c, double *scratch) {
    double acc[S_COUNT];
#pragma unroll
    for (int q = 0; q < S_COUNT; q++) acc[q] = 0.0;
    acc[S_NMIN] = INFINITY; acc[S_NHMIN] = INFINITY;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nquad; i += gridDim.x * blockDim.x) {
        const float4 h4 = __ldg(nH + i), n4 = __ldg(N + i), a4 = __ldg(Fx + i), b4 = __ldg(Fy + i), c4 = __ldg(Fz + i);
        const float4 x4 = __ldg(x + i), t4 = __ldg(T + i);
        const float h[4] = {h4.x, h4.y, h4.z, h4.w}, n[4] = {n4.x, n4.y, n4.z, n4.w};
        const float fx[4] = {a4.x, a4.y, a4.z, a4.w}, fy[4] = {b4.x, b4.y, b4.z, b4.w}, fz[4] = {c4.x, c4.y, c4.z, c4.w};
        const float xx[4] = {x4.x, x4.y, x4.z, x4.w}, tt[4] = {t4.x, t4.y, t4.z, t4.w};
#pragma unroll
        for (int q = 0; q < 4; q++) {
            const double hd = h[q];
            acc[S_M] += hd;
            acc[S_NHMIN] = fmin(acc[S_NHMIN], hd);
            acc[S_X] += xx[q];
            acc[S_XM] += hd * xx[q];
            acc[S_N] += n[q];
            acc[S_NM] += hd * n[q];
            acc[S_T] += tt[q];
            if (n[q] > 0.0f) {       // f = |F| / (c N)
                const double s = inv_c / n[q];
                const double rx = fx[q] * s, ry = fy[q] * s, rz = fz[q] * s;
                acc[S_F2MAX] = fmax(acc[S_F2MAX], rx * rx + ry * ry + rz * rz);
            }
            acc[S_NMIN] = fmin(acc[S_NMIN], (double)n[q]);
            const float chk = n[q] + fx[q] + fy[q] + fz[q] + xx[q] + tt[q];     // NaN/Inf poisons the sum
            if (!isfinite(n[q]) || !isfinite(fx[q]) || !isfinite(fy[q]) || !isfinite(fz[q]) || !isfinite(xx[q]) ||
                !isfinite(tt[q]) || chk != chk) acc[S_BAD] += 1.0;
            if (xx[q] >= 0.5f) acc[S_HALF] += 1.0;
        }
    }
    __shared__ double sh[8][S_COUNT];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < S_COUNT; q++) {
        const double v = is_max_row(q) ? wmax(acc[q]) : is_min_row(q) ? wmin(acc[q]) : wsum(acc[q]);
        if (lane == 0) sh[w][q] = v;
    }
    __syncthreads();
    if (threadIdx.x < S_COUNT) {
        const int q = threadIdx.x;
        double v = sh[0][q];
        for (int i = 1; i < 8; i++) v = is_max_row(q) ? fmax(v, sh[i][q]) : is_min_row(q) ? fmin(v, sh[i][q]) : v + sh[i][q];
        scratch[(size_t)blockIdx.x * S_COUNT + q] = v;
    }
}

// pass 2: one block sums rows [0, nrows) in a fixed order and writes the caller's sums in aton_reduce_sums' order
__global__ void __launch_bounds__(32) noalloc_pass2(const double *scratch, int nrows, double ncell, double *out) {
    const int q = threadIdx.x;
    double v = 0.0;
    if (q < S_COUNT) {
        v = scratch[q];
        for (int r = 1; r < nrows; r++) {
            const double p = scratch[(size_t)r * S_COUNT + q];
            v = is_max_row(q) ? fmax(v, p) : is_min_row(q) ? fmin(v, p) : v + p;
        }
    }
    // gather the rows in lane 0's order: [0] cells [1] sum x [2] sum nH x [3] sum nH [4] sum N [5] sum nH N [6] sum T
    // [7] cells with x >= 0.5 [8] non-finite cells [9] max f [10] min N [11] min nH
    const int src[ATON_NOALLOC_NSUMS] = {-1, S_X, S_XM, S_M, S_N, S_NM, S_T, S_HALF, S_BAD, S_F2MAX, S_NMIN, S_NHMIN};
    const int from = (q < ATON_NOALLOC_NSUMS && src[q < ATON_NOALLOC_NSUMS ? q : 0] >= 0) ? src[q] : 0;
    const double r = __shfl_sync(0xffffffffu, v, from);       // every lane takes part
    if (q < ATON_NOALLOC_NSUMS) out[q] = q == 0 ? ncell : (q == 9 ? sqrt(r) : r);
}

}  // namespace

extern "C" int aton_field_sums_noalloc(const float *nH, const float *x, const float *T, const float *N, const float *Fx,
                                       const float *Fy, const float *Fz, long long ncell, double c_cm_s, void *cuda_stream,
                                       double *sums) {
    using aton::fail;
    if (!nH || !x || !T || !N || !Fx || !Fy || !Fz || !sums)
        return fail(nullptr, ATON_EINVAL, "aton_field_sums_noalloc: NULL argument");
    if (ncell < 4 || ncell % 4 != 0)
        return fail(nullptr, ATON_EINVAL, "aton_field_sums_noalloc: ncell = %lld must be a positive multiple of 4", ncell);
    if (ncell > NOALLOC_MAX_CELLS)
        return fail(nullptr, ATON_EINVAL, "aton_field_sums_noalloc: ncell = %lld exceeds the maximum of %lld cells", ncell,
                    NOALLOC_MAX_CELLS);
    const float *ptrs[7] = {nH, x, T, N, Fx, Fy, Fz};
    for (const float *p : ptrs)
        if (reinterpret_cast<std::uintptr_t>(p) % 16 != 0)
            return fail(nullptr, ATON_EINVAL, "aton_field_sums_noalloc: the field arrays must be 16-byte aligned");
    const double c = c_cm_s > 0.0 ? c_cm_s : 2.99792458e10;
    int dev = -1;
    CU(nullptr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES)
        return fail(nullptr, ATON_EINVAL, "aton_field_sums_noalloc: device %d is beyond the %d this entry point serves", dev, MAX_DEVICES);
    if (!g_scratch_addr[dev]) {          // once per device, that device current: the array's DEVICE address
        double *p = nullptr;
        CU(nullptr, cudaGetSymbolAddress((void **)&p, g_noalloc_scratch));
        if (!p) return fail(nullptr, ATON_ECUDA, "aton_field_sums_noalloc: cudaGetSymbolAddress gave no address");
        g_scratch_addr[dev] = p;
    }
    double *scratch = g_scratch_addr[dev];
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int nquad = (int)(ncell / 4);
    const int blocks = std::min((nquad + 255) / 256, NOALLOC_ROWS);
    noalloc_pass1<<<blocks, 256, 0, stream>>>((const float4 *)N, (const float4 *)Fx, (const float4 *)Fy, (const float4 *)Fz,
                                              (const float4 *)x, (const float4 *)T, (const float4 *)nH, nquad, 1.0 / c, scratch);
    CU(nullptr, cudaGetLastError());
    noalloc_pass2<<<1, 32, 0, stream>>>(scratch, blocks, (double)ncell, sums);
    CU(nullptr, cudaGetLastError());
    return ATON_OK;
}
