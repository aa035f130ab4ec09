// Fused step kernel, variant 2: the FALLBACK for grids the product kernel (variant 4, aton_step_v4.cuh) cannot tile
// (nx % 32 != 0 or ny % 4 != 0) and the home of the Quad / flux_row helpers variant 4 shares.  Transport + injection +
// chemistry in one pass that reads every (N, G) value from HBM once (profiles/r01_b_step_fused_512.md).
//
// Decomposition:
//  * one WARP per tile row of 128 cells: lane l owns the quad of cells 4l..4l+3 (one 128-bit access per
//    field), held as two f2 pairs so that the arithmetic runs on FFMA2/FADD2/FMUL2 (aton_pk.cuh);
//  * a CTA is TY own rows plus one halo row below and one above (TY+2 warps) and marches through a
//    z-chunk of `lz` planes plus one halo plane on each side;
//  * every thread stages its own quad of the next plane with cp.async (double buffered, private to the
//    thread: no barrier protects it); the two edge lanes of a row also stage the x-halo cell;
//  * per staged cell the M1 closure is evaluated once; with U = (N,Gx,Gy,Gz), F_d = (G_d, P_dx, P_dy, P_dz)
//    the Lax-Friedrichs update (oracle O2) is
//        U' = (1 - 6h) U + h * sum_d [ (U + F_d)(i - e_d) + (U - F_d)(i + e_d) ],  h = c dt / (2 dx):
//      z: (U -+ F_z) never leave registers (the plane below waits one iteration for its +z term);
//      x: (U +- F_x) of the neighbouring quads come from warp shuffles;
//      y: each row publishes (U + F_y) and (U - F_y) once to shared memory (double buffered, one
//         __syncthreads per plane), the halo warps publish theirs and do nothing else;
//  * a finished cell goes through source injection and ONE chemistry sub-step over dt (chem_fast2);
//    cells that need sub-cycling are flagged in a bit mask and redone by step_fixup_kernel.
// Algorithmic traffic: 7 reads + 6 writes of fp32 per cell-update = 52 B.
#pragma once
#include "aton_async.cuh"
#include "aton_physics_pk.cuh"
#include "aton_step_ref.cuh"

namespace aton {

template <int TY>
struct FusedCfg {
    static constexpr int ROWS = TY + 2, THREADS = 32 * ROWS;
    static constexpr int RS = 136;                       // raw row: own quads at col 4.., x halos at 3 and 4+4*txn
    static constexpr int RAW_FIELD = ROWS * RS;
    static constexpr int RAW_BUF = 4 * RAW_FIELD;        // [field][row][RS]
    static constexpr int W_COMP = TY * 128;              // plus: staged rows 0..TY-1, minus: rows 2..TY+1
    static constexpr int W_BUF = 2 * 4 * W_COMP;         // [sign][comp][row][128]
    static constexpr size_t SMEM = (size_t)(2 * RAW_BUF + 2 * W_BUF) * sizeof(float);
};

struct Quad {           // 4 x-adjacent cells as two pairs, per conserved variable
    f2 v[2][4];         // [pair][N, Gx, Gy, Gz]
};

__device__ __forceinline__ f2 ld_pair(const float4 &q, int p) { return p == 0 ? pk(q.x, q.y) : pk(q.z, q.w); }

// flux rows of a pair: F_d = (G_d, P_dx, P_dy, P_dz) with P_dj = a delta_dj + s G_d G_j
__device__ __forceinline__ void flux_row(int d, const f2 u[4], f2 a, f2 s, f2 F[4]) {
    const f2 t = s * u[1 + d];
    F[0] = u[1 + d];
    F[1] = d == 0 ? fma2(t, u[1], a) : t * u[1];
    F[2] = d == 1 ? fma2(t, u[2], a) : t * u[2];
    F[3] = d == 2 ? fma2(t, u[3], a) : t * u[3];
}

template <int FLAGS, int TY>
__global__ void __launch_bounds__(32 * (TY + 2), (TY <= 8 ? 2 : 1))
step_fused_kernel(FieldsIO f, Grid g, StepConst c, int lz) {
    using C = FusedCfg<TY>;
    extern __shared__ __align__(16) float smem[];
    float *raw = smem;                       // [2][4][ROWS][RS]
    float *wy = smem + 2 * C::RAW_BUF;       // [2][2][4][TY][128]

    const int lane = threadIdx.x & 31, row = threadIdx.x >> 5;
    const int nq = g.nx >> 2;
    const int q0 = blockIdx.x * 32, j0 = blockIdx.y * TY, z0 = blockIdx.z * lz;
    const int txn = min(32, nq - q0), tyn = min(TY, g.ny - j0), lzn = min(lz, g.nz - z0);
    const bool lane_on = lane < txn;
    const bool own = row >= 1 && row <= tyn;
    const bool halo = row == 0 || row == tyn + 1;
    const bool edge_l = own && lane == 0, edge_r = own && lane == txn - 1;
    int j = j0 - 1 + row;
    j += j < 0 ? g.ny : 0;
    j -= j >= g.ny ? g.ny : 0;
    const int i = 4 * (q0 + lane);
    const int im = q0 == 0 ? g.nx - 1 : 4 * q0 - 1;
    const int ip = 4 * (q0 + txn) == g.nx ? 0 : 4 * (q0 + txn);
    const int plane = g.nx * g.ny;
    const int rowoff = j * g.nx;
    const float *src[4] = {f.N, f.Gx, f.Gy, f.Gz};
    const int my = row * C::RS + 4 + 4 * lane;           // own quad inside a raw field

    auto plane_of = [&](int m) {
        int k = z0 - 1 + m;
        k += k < 0 ? g.nz : 0;
        k -= k >= g.nz ? g.nz : 0;
        return k;
    };
    auto stage = [&](int m) {
        const bool inpl = m >= 1 && m <= lzn;
        float *dst = raw + (m & 1) * C::RAW_BUF;
        const int base = plane_of(m) * plane + rowoff;
        if (lane_on && (own || (halo && inpl))) {
#pragma unroll
            for (int v = 0; v < 4; v++) cp_async16(dst + v * C::RAW_FIELD + my, src[v] + base + i);
        }
        if (inpl && edge_l) {
#pragma unroll
            for (int v = 0; v < 4; v++) cp_async4(dst + v * C::RAW_FIELD + row * C::RS + 3, src[v] + base + im);
        }
        if (inpl && edge_r) {
#pragma unroll
            for (int v = 0; v < 4; v++)
                cp_async4(dst + v * C::RAW_FIELD + row * C::RS + 4 + 4 * txn, src[v] + base + ip);
        }
        cp_async_commit();
    };

    const f2 zero = splat(0.0f);
    Quad pend, zup;          // plane m-1 awaiting its +z term; h*(U + F_z) of plane m-1
#pragma unroll
    for (int p = 0; p < 2; p++)
#pragma unroll
        for (int v = 0; v < 4; v++) { pend.v[p][v] = zero; zup.v[p][v] = zero; }

    stage(0);
    for (int m = 0; m <= lzn + 1; m++) {
        cp_async_wait_all();                            // this thread's part of plane m has landed
        if (m + 1 <= lzn + 1) stage(m + 1);
        const bool inpl = m >= 1 && m <= lzn;
        const float *buf = raw + (m & 1) * C::RAW_BUF;
        float *wp = wy + (m & 1) * C::W_BUF;             // [0]: plus rows, [1]: minus rows
        float *wm = wp + 4 * C::W_COMP;

        // early loads for the chemistry of plane m-1
        const int oprev = plane_of(m - 1) * plane + rowoff + i;
        const bool fin = own && lane_on && m >= 2;
        float4 x4 = make_float4(0.f, 0.f, 0.f, 0.f), T4 = x4, h4 = make_float4(1.f, 1.f, 1.f, 1.f);
        bool has_src = false;
        if (fin) {
            x4 = *reinterpret_cast<const float4 *>(f.x + oprev);
            T4 = *reinterpret_cast<const float4 *>(f.T + oprev);
            h4 = __ldg(reinterpret_cast<const float4 *>(f.nH + oprev));
            has_src = source_segment_flag(f, oprev);
        }

        // ---- phase A: closure of the staged row, publish y terms, z terms, x terms
        const bool work = (own || (halo && inpl)) && row <= tyn + 1;
        Quad cur;
        f2 Sx[2][4];                 // (U + F_x)(i-1) + (U - F_x)(i+1) per own cell
        if (work) {
            Quad u;
            f2 a[2], s[2];
            {
                const float4 n4 = *reinterpret_cast<const float4 *>(buf + my);
                const float4 gx4 = *reinterpret_cast<const float4 *>(buf + C::RAW_FIELD + my);
                const float4 gy4 = *reinterpret_cast<const float4 *>(buf + 2 * C::RAW_FIELD + my);
                const float4 gz4 = *reinterpret_cast<const float4 *>(buf + 3 * C::RAW_FIELD + my);
#pragma unroll
                for (int p = 0; p < 2; p++) {
                    u.v[p][0] = ld_pair(n4, p); u.v[p][1] = ld_pair(gx4, p);
                    u.v[p][2] = ld_pair(gy4, p); u.v[p][3] = ld_pair(gz4, p);
                    closure2(u.v[p][0], u.v[p][1], u.v[p][2], u.v[p][3], a[p], s[p]);
                }
            }
            if (inpl) {
                // y: publish (U + F_y) for the row above, (U - F_y) for the row below
                const bool pub_p = row + 1 <= tyn, pub_m = row >= 2;
                f2 F[2][4];
                flux_row(1, u.v[0], a[0], s[0], F[0]);
                flux_row(1, u.v[1], a[1], s[1], F[1]);
#pragma unroll
                for (int v = 0; v < 4; v++) {
                    if (pub_p) {
                        const f2 w0 = u.v[0][v] + F[0][v], w1 = u.v[1][v] + F[1][v];
                        *reinterpret_cast<float4 *>(wp + v * C::W_COMP + row * 128 + 4 * lane) = make_float4(lo(w0), hi(w0), lo(w1), hi(w1));
                    }
                    if (pub_m) {
                        const f2 w0 = u.v[0][v] - F[0][v], w1 = u.v[1][v] - F[1][v];
                        *reinterpret_cast<float4 *>(wm + v * C::W_COMP + (row - 2) * 128 + 4 * lane) = make_float4(lo(w0), hi(w0), lo(w1), hi(w1));
                    }
                }
            }
            if (own) {
                // z: complete plane m-1, start plane m, seed plane m+1
#pragma unroll
                for (int p = 0; p < 2; p++) {
                    f2 F[4];
                    flux_row(2, u.v[p], a[p], s[p], F);
#pragma unroll
                    for (int v = 0; v < 4; v++) {
                        pend.v[p][v] = fma2(u.v[p][v] - F[v], c.h, pend.v[p][v]);
                        cur.v[p][v] = fma2(u.v[p][v], c.keep, zup.v[p][v]);
                        zup.v[p][v] = (u.v[p][v] + F[v]) * c.h;
                    }
                }
            }
            if (own && inpl) {
                // x: (U + F_x) of the cell to the left, (U - F_x) of the cell to the right
                f2 Wp[2][4], Wm[2][4];
#pragma unroll
                for (int p = 0; p < 2; p++) {
                    f2 F[4];
                    flux_row(0, u.v[p], a[p], s[p], F);
#pragma unroll
                    for (int v = 0; v < 4; v++) { Wp[p][v] = u.v[p][v] + F[v]; Wm[p][v] = u.v[p][v] - F[v]; }
                }
                f2 eWp[4], eWm[4];
#pragma unroll
                for (int v = 0; v < 4; v++) { eWp[v] = zero; eWm[v] = zero; }
                if (edge_l || edge_r) {      // pair (left halo cell, right halo cell) through the same formulas
                    const int cl = row * C::RS + 3, cr = row * C::RS + 4 + 4 * txn;
                    f2 e[4], ea, es, F[4];
#pragma unroll
                    for (int v = 0; v < 4; v++)      // a lane uses only the half it staged itself
                        e[v] = pk(buf[v * C::RAW_FIELD + cl], buf[v * C::RAW_FIELD + cr]);
                    closure2(e[0], e[1], e[2], e[3], ea, es);
                    flux_row(0, e, ea, es, F);
#pragma unroll
                    for (int v = 0; v < 4; v++) { eWp[v] = e[v] + F[v]; eWm[v] = e[v] - F[v]; }
                }
#pragma unroll
                for (int v = 0; v < 4; v++) {
                    float left = __shfl_up_sync(0xffffffffu, hi(Wp[1][v]), 1);
                    float right = __shfl_down_sync(0xffffffffu, lo(Wm[0][v]), 1);
                    if (edge_l) left = lo(eWp[v]);
                    if (edge_r) right = hi(eWm[v]);
                    Sx[0][v] = pk(left + hi(Wm[0][v]), lo(Wp[0][v]) + lo(Wm[1][v]));
                    Sx[1][v] = pk(hi(Wp[0][v]) + hi(Wm[1][v]), lo(Wp[1][v]) + right);
                }
            }
        }
        if (inpl) __syncthreads();                      // every row of the plane has published (uniform)
        // ---- phase B: y terms from shared memory
        if (own && inpl) {
            const int rp = (row - 1) * 128 + 4 * lane;
#pragma unroll
            for (int v = 0; v < 4; v++) {
                const float4 yp = *reinterpret_cast<const float4 *>(wp + v * C::W_COMP + rp);
                const float4 ym = *reinterpret_cast<const float4 *>(wm + v * C::W_COMP + rp);
#pragma unroll
                for (int p = 0; p < 2; p++) {
                    const f2 sxy = Sx[p][v] + (ld_pair(yp, p) + ld_pair(ym, p));
                    cur.v[p][v] = fma2(sxy, c.h, cur.v[p][v]);
                }
            }
        }

        // plane m-1 has all six contributions: inject, one chemistry sub-step, store
        if (fin) {
            if (has_src) {
                pend.v[0][0] = pend.v[0][0] + pk(source_lookup(f, oprev, c.dt), source_lookup(f, oprev + 1, c.dt));
                pend.v[1][0] = pend.v[1][0] + pk(source_lookup(f, oprev + 2, c.dt), source_lookup(f, oprev + 3, c.dt));
            }
            f2 xs[2] = {pk(x4.x, x4.y), pk(x4.z, x4.w)}, Ts[2] = {pk(T4.x, T4.y), pk(T4.z, T4.w)};
            const f2 hs[2] = {pk(h4.x, h4.y), pk(h4.z, h4.w)};
            unsigned nib = 0;
#pragma unroll
            for (int p = 0; p < 2; p++)
                nib |= chem_fast2<FLAGS>(pend.v[p][0], pend.v[p][1], pend.v[p][2], pend.v[p][3], xs[p], Ts[p], hs[p], c)
                       << (2 * p);
#define ATON_ST4(ptr, A, B) *reinterpret_cast<float4 *>(ptr + oprev) = make_float4(lo(A), hi(A), lo(B), hi(B))
            ATON_ST4(f.N1, pend.v[0][0], pend.v[1][0]);
            ATON_ST4(f.Gx1, pend.v[0][1], pend.v[1][1]);
            ATON_ST4(f.Gy1, pend.v[0][2], pend.v[1][2]);
            ATON_ST4(f.Gz1, pend.v[0][3], pend.v[1][3]);
            ATON_ST4(f.x, xs[0], xs[1]);
            ATON_ST4(f.T, Ts[0], Ts[1]);
#undef ATON_ST4
            if (nib) atomicOr(f.defer_mask + ((unsigned)oprev >> 5), nib << (oprev & 31));
        }
        if (own) pend = cur;
    }
}

inline int fused_default_lz(const Grid &g, int ty, int tile_z) {
    if (tile_z > 0) return tile_z < g.nz ? tile_z : g.nz;
    const long tiles_xy = (long)((g.nx / 4 + 31) / 32) * ((g.ny + ty - 1) / ty);
    int lz = 64;      // largest power of two <= 64 that still gives >= 4 CTAs per SM
    while (lz > 4 && tiles_xy * ((g.nz + lz - 1) / lz) < 4L * 148) lz >>= 1;
    return lz < g.nz ? lz : g.nz;
}

template <int FLAGS, int TY>
cudaError_t launch_step_fused_ty(const FieldsIO &f, const Grid &g, const StepConst &c, int tile_z, cudaStream_t stream) {
    using C = FusedCfg<TY>;
    // per device, not per process: set it at every launch (a cheap driver call)
    cudaError_t e = cudaFuncSetAttribute(step_fused_kernel<FLAGS, TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    const int lz = fused_default_lz(g, TY, tile_z);
    const dim3 grid((g.nx / 4 + 31) / 32, (g.ny + TY - 1) / TY, (g.nz + lz - 1) / lz);
    step_fused_kernel<FLAGS, TY><<<grid, C::THREADS, C::SMEM, stream>>>(f, g, c, lz);
    return cudaGetLastError();
}

inline bool fused_shape_ok(int tile_y, int tile_z) {
    return (tile_y == 0 || tile_y == 6 || tile_y == 14) && tile_z >= 0;
}

// one step = fused kernel, then (when the physics can sub-cycle, i.e. cooling is on) the fix-up kernel (aton_fixup.cuh)
template <int FLAGS>
cudaError_t launch_step_fused(const FieldsIO &f, const Grid &g, const StepConst &c, int tile_y, int tile_z,
                              cudaStream_t stream) {
    if (tile_y == 14) return launch_step_fused_ty<FLAGS, 14>(f, g, c, tile_z, stream);
    return launch_step_fused_ty<FLAGS, 6>(f, g, c, tile_z, stream);    // default: measured fastest
}

}  // namespace aton
