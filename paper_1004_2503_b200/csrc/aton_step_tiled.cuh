// Tiled streaming step kernel (variant 1, the product kernel): fused transport + injection + chemistry
// that reads every (N, G) value from HBM once.
//
// Decomposition:
//  * a CTA owns an x-y tile of TXQ quads (4 cells, one 128-bit access) by TY rows and marches through a
//    z-chunk of LZ planes (plus one halo plane on each side);
//  * the next plane's (N, Gx, Gy, Gz) tile, with its one-cell x/y halo (periodic wrap resolved in the
//    source address), is staged into shared memory with cp.async while the current plane is computed
//    (double buffered, no register staging);
//  * the M1 closure is evaluated once per staged cell (own cells and halo cells), published as (a, s)
//    in shared memory, and the 7-point Lax-Friedrichs update is assembled as a sum of neighbour
//    contributions: x/y neighbours are read from shared memory, z neighbours never leave registers
//    (each plane adds its "down" contribution to the pending plane below and seeds the plane above);
//  * when a plane has all six contributions the cell goes straight through source injection and the
//    sub-cycled chemistry in registers and is written out: N, G to the other ping-pong buffer, x and T
//    in place.  Algorithmic traffic: 7 reads + 6 writes of fp32 per cell-update = 52 B.
#pragma once
#include "aton_step_ref.cuh"

namespace aton {

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem, const void *gmem) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

struct TileShape {
    int txq, ty, lz;     // quads per tile row, rows per tile, planes per z-chunk
};

// shared-memory footprint: 2 raw buffers x 4 fields + (a, s), each (ty+2) rows of (4 txq + 8) floats
inline size_t tiled_smem_bytes(const TileShape &t) {
    return (size_t)10 * (t.ty + 2) * (4 * t.txq + 8) * sizeof(float);
}

inline TileShape tiled_default_shape(const Grid &g, int tile_y, int tile_z) {
    TileShape t;
    const int nq = g.nx / 4;
    t.txq = nq < 32 ? nq : 32;
    t.ty = tile_y > 0 ? tile_y : 8;
    if (t.ty > g.ny) t.ty = g.ny;
    const long tiles_xy = (long)((nq + t.txq - 1) / t.txq) * ((g.ny + t.ty - 1) / t.ty);
    if (tile_z > 0) {
        t.lz = tile_z;
    } else {   // largest power of two <= 64 that still gives >= 4 CTAs per SM
        t.lz = 64;
        while (t.lz > 4 && tiles_xy * ((g.nz + t.lz - 1) / t.lz) < 4L * 148) t.lz >>= 1;
    }
    if (t.lz > g.nz) t.lz = g.nz;
    return t;
}

inline bool tiled_shape_ok(const Grid &g, int tile_y, int tile_z) {
    if (tile_y < 0 || tile_z < 0) return false;
    const TileShape t = tiled_default_shape(g, tile_y, tile_z);
    return t.txq * t.ty <= 512 && t.txq * t.ty >= 1 && tiled_smem_bytes(t) <= 200 * 1024;
}

// contribution of an x- or y-neighbour read from shared memory (same algebra as add_neighbour)
template <int D>
__device__ __forceinline__ void add_nb(float h, float sgn, float Nn, float gx, float gy, float gz, float a, float s,
                                       float &aN, float &ax, float &ay, float &az) {
    const float gd = D == 0 ? gx : (D == 1 ? gy : gz);
    const float t = s * gd;
    float px = t * gx, py = t * gy, pz = t * gz;
    if (D == 0) px += a; else if (D == 1) py += a; else pz += a;
    aN = fmaf(h, Nn - sgn * gd, aN);
    ax = fmaf(h, gx - sgn * px, ax);
    ay = fmaf(h, gy - sgn * py, ay);
    az = fmaf(h, gz - sgn * pz, az);
}

template <int FLAGS, int MAXT, int MINB>
__device__ __forceinline__ void step_tiled_body(const FieldsIO &f, const Grid &g, const StepConst &c, const TileShape &ts) {
    extern __shared__ __align__(16) float smem[];
    const int RS = 4 * ts.txq + 8;                 // row stride (floats); own quads start at column 4
    const int PL = (ts.ty + 2) * RS;               // floats per array
    float *raw = smem;                             // [2][4][PL]
    float *sa = smem + 8 * PL, *ss = smem + 9 * PL;

    const int tx = threadIdx.x, ty = threadIdx.y;
    const int tid = ty * ts.txq + tx, nthr = ts.txq * ts.ty;
    const int nq = g.nx >> 2;
    const int q0 = blockIdx.x * ts.txq, j0 = blockIdx.y * ts.ty, z0 = blockIdx.z * ts.lz;
    const int txn = min(ts.txq, nq - q0), tyn = min(ts.ty, g.ny - j0), lzn = min(ts.lz, g.nz - z0);
    const bool active = tx < txn && ty < tyn;
    const int i = 4 * (q0 + tx), j = j0 + ty;
    const int plane = g.nx * g.ny;
    const int own = (ty + 1) * RS + 4 + 4 * tx;    // smem offset of the own quad
    // halo geometry (periodic wrap resolved here)
    const int jm = (j0 - 1 + g.ny) % g.ny, jp = (j0 + tyn) % g.ny;
    const int im = (4 * q0 - 1 + g.nx) % g.nx, ip = (4 * (q0 + txn)) % g.nx;
    const int n_items = 2 * txn + 2 * tyn;         // 2 halo rows of quads, then 2 halo columns of cells

    auto plane_of = [&](int m) { return (z0 - 1 + m + g.nz) % g.nz; };

    auto stage = [&](int m) {                      // cp.async plane m into raw[m&1]
        const int kz = plane_of(m);
        float *dst = raw + (m & 1) * 4 * PL;
        const float *src[4] = {f.N, f.Gx, f.Gy, f.Gz};
        const size_t base = (size_t)kz * plane;
        if (active) {
            const size_t o = base + (size_t)j * g.nx + i;
#pragma unroll
            for (int v = 0; v < 4; v++) cp_async16(dst + v * PL + own, src[v] + o);
        }
        for (int it = tid; it < n_items; it += nthr) {
            if (it < 2 * txn) {
                const int hi = it >= txn, q = it - hi * txn;
                const size_t o = base + (size_t)(hi ? jp : jm) * g.nx + 4 * (q0 + q);
                const int so = (hi ? tyn + 1 : 0) * RS + 4 + 4 * q;
#pragma unroll
                for (int v = 0; v < 4; v++) cp_async16(dst + v * PL + so, src[v] + o);
            } else {
                const int e = it - 2 * txn, hi = e >= tyn, r = e - hi * tyn;
                const size_t o = base + (size_t)(j0 + r) * g.nx + (hi ? ip : im);
                const int so = (r + 1) * RS + (hi ? 4 + 4 * txn : 3);
#pragma unroll
                for (int v = 0; v < 4; v++) cp_async4(dst + v * PL + so, src[v] + o);
            }
        }
        cp_async_commit();
    };

    // accumulators of the plane awaiting its "down" contribution (A0) and of the current plane (A1)
    float A0[4][4], A1[4][4];
#pragma unroll
    for (int q = 0; q < 4; q++)
#pragma unroll
        for (int v = 0; v < 4; v++) { A0[q][v] = 0.f; A1[q][v] = 0.f; }
    int nsub_sum = 0, nsub_max = 0;

    stage(0);
    for (int m = 0; m <= lzn + 1; m++) {
        cp_async_wait_all();
        __syncthreads();                           // S1: plane m staged; previous in-plane reads done
        if (m + 1 <= lzn + 1) stage(m + 1);
        const float *buf = raw + (m & 1) * 4 * PL;
        const int kprev = plane_of(m - 1);
        const size_t oprev = (size_t)kprev * plane + (size_t)j * g.nx + i;
        // early loads of the cell state needed by the chemistry of plane m-1
        float4 x4 = make_float4(0, 0, 0, 0), T4 = x4, h4 = x4;
        const bool fin = active && m >= 2;
        if (fin) {
            x4 = *reinterpret_cast<const float4 *>(f.x + oprev);
            T4 = *reinterpret_cast<const float4 *>(f.T + oprev);
            h4 = __ldg(reinterpret_cast<const float4 *>(f.nH + oprev));
        }
        // closure once per staged cell: own quad ...
        float A2[4][4];
        if (active) {
            const float4 n4 = *reinterpret_cast<const float4 *>(buf + own);
            const float4 gx4 = *reinterpret_cast<const float4 *>(buf + PL + own);
            const float4 gy4 = *reinterpret_cast<const float4 *>(buf + 2 * PL + own);
            const float4 gz4 = *reinterpret_cast<const float4 *>(buf + 3 * PL + own);
            const float Nq[4] = {n4.x, n4.y, n4.z, n4.w}, X[4] = {gx4.x, gx4.y, gx4.z, gx4.w};
            const float Y[4] = {gy4.x, gy4.y, gy4.z, gy4.w}, Z[4] = {gz4.x, gz4.y, gz4.z, gz4.w};
            float a[4], s[4];
#pragma unroll
            for (int q = 0; q < 4; q++) {
                closure(Nq[q], X[q], Y[q], Z[q], a[q], s[q]);
                // z-neighbour contributions stay in registers: P_zj = a delta_zj + s Gz Gj
                const float t = s[q] * Z[q];
                const float pzx = t * X[q], pzy = t * Y[q], pzz = fmaf(t, Z[q], a[q]);
                // "down": this plane is the +z neighbour of plane m-1
                A0[q][0] = fmaf(c.h, Nq[q] - Z[q], A0[q][0]);
                A0[q][1] = fmaf(c.h, X[q] - pzx, A0[q][1]);
                A0[q][2] = fmaf(c.h, Y[q] - pzy, A0[q][2]);
                A0[q][3] = fmaf(c.h, Z[q] - pzz, A0[q][3]);
                // own term of this plane
                A1[q][0] = fmaf(c.keep, Nq[q], A1[q][0]);
                A1[q][1] = fmaf(c.keep, X[q], A1[q][1]);
                A1[q][2] = fmaf(c.keep, Y[q], A1[q][2]);
                A1[q][3] = fmaf(c.keep, Z[q], A1[q][3]);
                // "up": this plane is the -z neighbour of plane m+1
                A2[q][0] = c.h * (Nq[q] + Z[q]);
                A2[q][1] = c.h * (X[q] + pzx);
                A2[q][2] = c.h * (Y[q] + pzy);
                A2[q][3] = c.h * (Z[q] + pzz);
            }
            *reinterpret_cast<float4 *>(sa + own) = make_float4(a[0], a[1], a[2], a[3]);
            *reinterpret_cast<float4 *>(ss + own) = make_float4(s[0], s[1], s[2], s[3]);
        }
        // ... and the halo cells (only planes of the chunk need in-plane neighbours)
        const bool inplane = m >= 1 && m <= lzn;
        if (inplane) {
            for (int it = tid; it < n_items; it += nthr) {
                if (it < 2 * txn) {
                    const int hi = it >= txn, q = it - hi * txn;
                    const int so = (hi ? tyn + 1 : 0) * RS + 4 + 4 * q;
                    const float4 n4 = *reinterpret_cast<const float4 *>(buf + so);
                    const float4 gx4 = *reinterpret_cast<const float4 *>(buf + PL + so);
                    const float4 gy4 = *reinterpret_cast<const float4 *>(buf + 2 * PL + so);
                    const float4 gz4 = *reinterpret_cast<const float4 *>(buf + 3 * PL + so);
                    float4 a4, s4;
                    closure(n4.x, gx4.x, gy4.x, gz4.x, a4.x, s4.x);
                    closure(n4.y, gx4.y, gy4.y, gz4.y, a4.y, s4.y);
                    closure(n4.z, gx4.z, gy4.z, gz4.z, a4.z, s4.z);
                    closure(n4.w, gx4.w, gy4.w, gz4.w, a4.w, s4.w);
                    *reinterpret_cast<float4 *>(sa + so) = a4;
                    *reinterpret_cast<float4 *>(ss + so) = s4;
                } else {
                    const int e = it - 2 * txn, hi = e >= tyn, r = e - hi * tyn;
                    const int so = (r + 1) * RS + (hi ? 4 + 4 * txn : 3);
                    float a1, s1;
                    closure(buf[so], buf[PL + so], buf[2 * PL + so], buf[3 * PL + so], a1, s1);
                    sa[so] = a1; ss[so] = s1;
                }
            }
        }
        __syncthreads();                           // S2: (a, s) of the whole staged tile visible
        if (active && inplane) {
            // y neighbours: quads of the rows above / below
#pragma unroll
            for (int side = 0; side < 2; side++) {
                const int o = own + (side ? RS : -RS);
                const float sgn = side ? 1.f : -1.f;
                const float4 n4 = *reinterpret_cast<const float4 *>(buf + o);
                const float4 gx4 = *reinterpret_cast<const float4 *>(buf + PL + o);
                const float4 gy4 = *reinterpret_cast<const float4 *>(buf + 2 * PL + o);
                const float4 gz4 = *reinterpret_cast<const float4 *>(buf + 3 * PL + o);
                const float4 a4 = *reinterpret_cast<const float4 *>(sa + o);
                const float4 s4 = *reinterpret_cast<const float4 *>(ss + o);
                add_nb<1>(c.h, sgn, n4.x, gx4.x, gy4.x, gz4.x, a4.x, s4.x, A1[0][0], A1[0][1], A1[0][2], A1[0][3]);
                add_nb<1>(c.h, sgn, n4.y, gx4.y, gy4.y, gz4.y, a4.y, s4.y, A1[1][0], A1[1][1], A1[1][2], A1[1][3]);
                add_nb<1>(c.h, sgn, n4.z, gx4.z, gy4.z, gz4.z, a4.z, s4.z, A1[2][0], A1[2][1], A1[2][2], A1[2][3]);
                add_nb<1>(c.h, sgn, n4.w, gx4.w, gy4.w, gz4.w, a4.w, s4.w, A1[3][0], A1[3][1], A1[3][2], A1[3][3]);
            }
            // x neighbours: the six cells own-1 .. own+4 of the own row
            float Nr[6], Xr[6], Yr[6], Zr[6], ar[6], sr[6];
            {
                const float4 n4 = *reinterpret_cast<const float4 *>(buf + own);
                const float4 gx4 = *reinterpret_cast<const float4 *>(buf + PL + own);
                const float4 gy4 = *reinterpret_cast<const float4 *>(buf + 2 * PL + own);
                const float4 gz4 = *reinterpret_cast<const float4 *>(buf + 3 * PL + own);
                const float4 a4 = *reinterpret_cast<const float4 *>(sa + own);
                const float4 s4 = *reinterpret_cast<const float4 *>(ss + own);
                Nr[1] = n4.x; Nr[2] = n4.y; Nr[3] = n4.z; Nr[4] = n4.w;
                Xr[1] = gx4.x; Xr[2] = gx4.y; Xr[3] = gx4.z; Xr[4] = gx4.w;
                Yr[1] = gy4.x; Yr[2] = gy4.y; Yr[3] = gy4.z; Yr[4] = gy4.w;
                Zr[1] = gz4.x; Zr[2] = gz4.y; Zr[3] = gz4.z; Zr[4] = gz4.w;
                ar[1] = a4.x; ar[2] = a4.y; ar[3] = a4.z; ar[4] = a4.w;
                sr[1] = s4.x; sr[2] = s4.y; sr[3] = s4.z; sr[4] = s4.w;
                const int l = own - 1, r = own + 4;
                Nr[0] = buf[l]; Xr[0] = buf[PL + l]; Yr[0] = buf[2 * PL + l]; Zr[0] = buf[3 * PL + l]; ar[0] = sa[l]; sr[0] = ss[l];
                Nr[5] = buf[r]; Xr[5] = buf[PL + r]; Yr[5] = buf[2 * PL + r]; Zr[5] = buf[3 * PL + r]; ar[5] = sa[r]; sr[5] = ss[r];
            }
#pragma unroll
            for (int q = 0; q < 4; q++) {
                add_nb<0>(c.h, -1.f, Nr[q], Xr[q], Yr[q], Zr[q], ar[q], sr[q], A1[q][0], A1[q][1], A1[q][2], A1[q][3]);
                add_nb<0>(c.h, 1.f, Nr[q + 2], Xr[q + 2], Yr[q + 2], Zr[q + 2], ar[q + 2], sr[q + 2], A1[q][0], A1[q][1], A1[q][2], A1[q][3]);
            }
        }
        // plane m-1 now has all six contributions: inject, chemistry, store
        if (fin) {
            float xs[4] = {x4.x, x4.y, x4.z, x4.w}, Ts[4] = {T4.x, T4.y, T4.z, T4.w};
            const float hs[4] = {h4.x, h4.y, h4.z, h4.w};
            if (source_segment_flag(f, (int)oprev)) {
#pragma unroll
                for (int q = 0; q < 4; q++) A0[q][0] += source_lookup(f, (int)oprev + q, c.dt);
            }
#pragma unroll
            for (int q = 0; q < 4; q++) {
                const int ns = chemistry<FLAGS>(A0[q][0], A0[q][1], A0[q][2], A0[q][3], xs[q], Ts[q], hs[q], c);
                nsub_sum += ns;
                nsub_max = max(nsub_max, ns);
            }
            *reinterpret_cast<float4 *>(f.N1 + oprev) = make_float4(A0[0][0], A0[1][0], A0[2][0], A0[3][0]);
            *reinterpret_cast<float4 *>(f.Gx1 + oprev) = make_float4(A0[0][1], A0[1][1], A0[2][1], A0[3][1]);
            *reinterpret_cast<float4 *>(f.Gy1 + oprev) = make_float4(A0[0][2], A0[1][2], A0[2][2], A0[3][2]);
            *reinterpret_cast<float4 *>(f.Gz1 + oprev) = make_float4(A0[0][3], A0[1][3], A0[2][3], A0[3][3]);
            *reinterpret_cast<float4 *>(f.x + oprev) = make_float4(xs[0], xs[1], xs[2], xs[3]);
            *reinterpret_cast<float4 *>(f.T + oprev) = make_float4(Ts[0], Ts[1], Ts[2], Ts[3]);
        }
        // rotate: current plane becomes the pending one; the "up" contribution seeds the next plane
#pragma unroll
        for (int q = 0; q < 4; q++)
#pragma unroll
            for (int v = 0; v < 4; v++) { A0[q][v] = A1[q][v]; A1[q][v] = active ? A2[q][v] : 0.f; }
    }

    // sub-cycle statistics: one atomic pair per CTA
    __shared__ int s_sum[32], s_max[32];
    int sum = nsub_sum, mx = nsub_max;
    for (int o = 16; o > 0; o >>= 1) {
        sum += __shfl_xor_sync(0xffffffffu, sum, o);
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((tid & 31) == 0) { s_sum[tid >> 5] = sum; s_max[tid >> 5] = mx; }
    __syncthreads();
    if (tid == 0) {
        const int nw = (nthr + 31) >> 5;
        for (int w = 1; w < nw; w++) { sum += s_sum[w]; mx = max(mx, s_max[w]); }
        atomicAdd(f.stats, (unsigned long long)sum);
        atomicMax(f.stats + 1, (unsigned long long)mx);
    }
}

// two register budgets: 256-thread tiles at 2 CTAs/SM (the 1024^3 configuration), anything else generic
template <int FLAGS>
__global__ void __launch_bounds__(256, 2) step_tiled_kernel_256(FieldsIO f, Grid g, StepConst c, TileShape ts) {
    step_tiled_body<FLAGS, 256, 2>(f, g, c, ts);
}
template <int FLAGS>
__global__ void __launch_bounds__(512, 1) step_tiled_kernel_512(FieldsIO f, Grid g, StepConst c, TileShape ts) {
    step_tiled_body<FLAGS, 512, 1>(f, g, c, ts);
}

template <int FLAGS>
cudaError_t launch_step_tiled(const FieldsIO &f, const Grid &g, const StepConst &c, int tile_y, int tile_z,
                              cudaStream_t stream) {
    const TileShape ts = tiled_default_shape(g, tile_y, tile_z);
    const int nq = g.nx / 4;
    const dim3 block(ts.txq, ts.ty, 1);
    const dim3 grid((nq + ts.txq - 1) / ts.txq, (g.ny + ts.ty - 1) / ts.ty, (g.nz + ts.lz - 1) / ts.lz);
    const size_t smem = tiled_smem_bytes(ts);
    static bool attr_done = false;     // one per FLAGS instantiation
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(step_tiled_kernel_256<FLAGS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(step_tiled_kernel_512<FLAGS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    if (ts.txq * ts.ty <= 256) step_tiled_kernel_256<FLAGS><<<grid, block, smem, stream>>>(f, g, c, ts);
    else step_tiled_kernel_512<FLAGS><<<grid, block, smem, stream>>>(f, g, c, ts);
    return cudaGetLastError();
}

}  // namespace aton
