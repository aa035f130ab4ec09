// Stand-alone probe (not part of libaton.so): which HBM throughput does the step kernel's ACCESS PATTERN allow?
// 7 fp32 arrays read + 6 written per cell (the 52 B of a cell-update) at 1024^3, no arithmetic, no halos; a warp
// owns a tile of WXQ quads x 32/WXQ rows and marches along z (or y) like step_v4_kernel.  Results on B200 and
// what they meant for the tile shape: profiles/r01_e_tile_shape.md.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o probe_tile_pattern probe_tile_pattern.cu && ./probe_tile_pattern
#include <cstdio>
#include <cuda_runtime.h>
struct P { const float4 *in[7]; float4 *out[6]; };
// lanes: q = lane % WXQ (quad in x), r = lane / WXQ (row); WXQ*WR == 32.  CTA = 4 warps side by side in x.
template <int WXQ, int MARCH_Y>
__global__ void __launch_bounds__(128) tiles(P p, int n, int lm) {
    constexpr int WR = 32 / WXQ;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, r = lane / WXQ, q = lane % WXQ;
    const int x0 = (blockIdx.x * 4 + warp) * WXQ * 4;
    const size_t rowq = n / 4, plane = (size_t)n * n / 4;
    size_t o, step;
    if (!MARCH_Y) { o = (size_t)(blockIdx.z * lm) * plane + (size_t)(blockIdx.y * WR + r) * rowq + x0 / 4 + q; step = plane; }
    else          { o = (size_t)(blockIdx.z * WR + r) * plane + (size_t)(blockIdx.y * lm) * rowq + x0 / 4 + q; step = rowq; }
    for (int k = 0; k < lm; k++, o += step) {
        float4 a[7];
#pragma unroll
        for (int f = 0; f < 7; f++) a[f] = p.in[f][o];
        float4 s = a[6];
#pragma unroll
        for (int f = 0; f < 6; f++) { float4 v = a[f]; v.x += s.x; v.y += s.y; v.z += s.z; v.w += s.w; p.out[f][o] = v; }
    }
}
// reference: the same 13 streams read / written in plain grid-stride order
__global__ void __launch_bounds__(256) mix(P p, size_t nq) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nq; i += (size_t)gridDim.x * blockDim.x) {
        float4 a[7];
#pragma unroll
        for (int k = 0; k < 7; k++) a[k] = p.in[k][i];
        float4 s = a[6];
#pragma unroll
        for (int k = 0; k < 6; k++) { float4 v = a[k]; v.x += s.x; v.y += s.y; v.z += s.z; v.w += s.w; p.out[k][i] = v; }
    }
}
template <int WXQ, int MARCH_Y>
void run(const char *name, P p, int n, int lm) {
    constexpr int WR = 32 / WXQ;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1); float ms;
    dim3 g(n / (16 * WXQ), MARCH_Y ? n / lm : n / WR, MARCH_Y ? n / WR : n / lm);
    tiles<WXQ, MARCH_Y><<<g, 128>>>(p, n, lm);
    cudaEventRecord(e0); for (int i = 0; i < 5; i++) tiles<WXQ, MARCH_Y><<<g, 128>>>(p, n, lm); cudaEventRecord(e1); cudaEventSynchronize(e1);
    cudaEventElapsedTime(&ms, e0, e1);
    printf("%-28s lm %4d: %.3f ms  %.0f GB/s  %s\n", name, lm, ms / 5, 13.0 * n * n * (double)n * 4 / (ms / 5 * 1e-3) / 1e9, cudaGetErrorString(cudaGetLastError()));
}
int main() {
    const int n = 1024; const size_t ne = (size_t)n * n * n;
    P p; float *buf[13];
    for (int k = 0; k < 13; k++) { cudaMalloc(&buf[k], ne * 4); cudaMemset(buf[k], 0, ne * 4); }
    for (int k = 0; k < 7; k++) p.in[k] = (const float4 *)buf[k];
    for (int k = 0; k < 6; k++) p.out[k] = (float4 *)buf[7 + k];
    {
        cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1); float ms;
        mix<<<148 * 16, 256>>>(p, ne / 4);
        cudaEventRecord(e0); for (int i = 0; i < 5; i++) mix<<<148 * 16, 256>>>(p, ne / 4); cudaEventRecord(e1); cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        printf("%-28s         : %.3f ms  %.0f GB/s\n", "7r + 6w, grid-stride", ms / 5, 13.0 * ne * 4 / (ms / 5 * 1e-3) / 1e9);
    }
    for (int lm : {16, 64, 256, 1024}) run<8, 0>("32x4 tile, march z", p, n, lm);
    for (int lm : {64, 256}) run<16, 0>("64x2 tile, march z", p, n, lm);
    for (int lm : {64, 256}) run<32, 0>("128x1 tile, march z", p, n, lm);
    for (int lm : {16, 64, 256, 1024}) run<8, 1>("32 x 4 planes, march y", p, n, lm);
    for (int lm : {64, 256}) run<32, 1>("128 x 1 plane, march y", p, n, lm);
    return 0;
}
