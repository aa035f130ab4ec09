// Fused step kernel, variant 3 (the product kernel for grids with nx % 128 == 0 and ny % TY == 0):
// transport + injection + one chemistry sub-step in one pass over HBM, 52 B per cell-update.
//
// Same arithmetic as variant 2 (aton_step_fused.cuh: packed fp32x2 pairs, closure once per staged cell,
// z terms in registers, x terms by warp shuffles, y terms through shared memory, sub-cycling cells
// deferred to step_fixup_kernel); only the order in which the x and y neighbour terms are summed differs,
// so results agree with variant 2 to rounding.  What changes is the
// execution shape, driven by profiles/r01_b_step_fused_512.md (issue slots 45 % busy, 3.2 of 9.4 warp
// states per issue at the CTA barrier, 2 of 8 warps idle halo warps):
//  * no halo warps: a CTA is TY warps = TY own rows; the first / last warp also stages the row below /
//    above the tile and publishes its y term (closure + F_y only), so every resident warp carries a full
//    row of work and the register file is not spent on idle warps;
//  * split-phase barrier: a warp publishes the y terms of plane m, ARRIVES on an mbarrier, then does
//    all the work that needs nobody else (z terms, x terms, injection + chemistry + stores of plane
//    m-1) and only then WAITS for the plane's y terms -- by then every warp has long arrived;
//  * the last accumulation writes the loop-carried registers directly (no register-to-register copies),
//    tiles are always full (no ragged-edge predicates) and plane offsets advance incrementally.
#pragma once
#include "aton_step_fused.cuh"

namespace aton {

template <int TY>
struct V3Cfg {
    static constexpr int ROWS = TY + 2, THREADS = 32 * TY;
    static constexpr int RS = 136;                       // raw row: own quads at col 4.., x halos at 3 and 132
    static constexpr int RAW_FIELD = ROWS * RS;
    static constexpr int RAW_BUF = 4 * RAW_FIELD;        // [field][row slot][RS]; slot 0 / TY+1 = y halo rows
    static constexpr int W_COMP = TY * 128;              // plus: slot r = (U+F_y) of row r-1; minus: slot r = row r+1
    static constexpr int W_BUF = 2 * 4 * W_COMP;         // [sign][comp][slot][128]
    static constexpr size_t SMEM = (size_t)(2 * RAW_BUF + 2 * W_BUF) * sizeof(float);
};

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned addr, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(addr), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned addr) {
    asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(addr) : "memory");
}
__device__ __forceinline__ bool mbar_try(unsigned addr, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.acquire.cta.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    return ok != 0;
}
#ifndef ATON_WAIT_SLEEP_NS
#define ATON_WAIT_SLEEP_NS 0
#endif
__device__ __forceinline__ void mbar_wait(unsigned addr, unsigned parity) {
    while (!mbar_try(addr, parity)) {
        if (ATON_WAIT_SLEEP_NS > 0) __nanosleep(ATON_WAIT_SLEEP_NS);
    }
}

template <int FLAGS, int TY>
__global__ void __launch_bounds__(32 * TY, (TY <= 8 ? 2 : 1))
step_v3_kernel(FieldsIO f, Grid g, StepConst c, int lz) {
    using C = V3Cfg<TY>;
    extern __shared__ __align__(16) float smem[];
    __shared__ __align__(8) unsigned long long bars[2];
    float *raw = smem;                       // [2][4][ROWS][RS]
    float *wy = smem + 2 * C::RAW_BUF;       // [2][2][4][TY][128]

    const int lane = threadIdx.x & 31, row = threadIdx.x >> 5;
    const int q0 = blockIdx.x * 32, j0 = blockIdx.y * TY, z0 = blockIdx.z * lz;
    const int lzn = min(lz, g.nz - z0);
    const bool bot = row == 0, top = row == TY - 1;
    const bool edge_l = lane == 0, edge_r = lane == 31;
    const int plane = g.nx * g.ny;
    const int i = 4 * (q0 + lane);
    const int im = q0 == 0 ? g.nx - 1 : 4 * q0 - 1;
    const int ip = 4 * (q0 + 32) == g.nx ? 0 : 4 * (q0 + 32);
    const int rowoff = (j0 + row) * g.nx;
    // y halo row staged by the first (row below the tile) / last (row above) warp
    const int jh = bot ? (j0 == 0 ? g.ny - 1 : j0 - 1) : (j0 + TY == g.ny ? 0 : j0 + TY);
    const int hrowoff = jh * g.nx;
    const int hslot = bot ? 0 : TY + 1;
    const float *src[4] = {f.N, f.Gx, f.Gy, f.Gz};
    const int my = (row + 1) * C::RS + 4 + 4 * lane;     // own quad inside a raw field
    const int myh = hslot * C::RS + 4 + 4 * lane;        // halo-row quad
    const unsigned bar0 = smem_u32(&bars[0]);

    if (threadIdx.x == 0) {
        mbar_init(bar0, TY);
        mbar_init(bar0 + 8, TY);
    }
    __syncthreads();

    // element offset of staged plane m = z0 - 1 + m (periodic); advanced incrementally
    int kst = z0 == 0 ? g.nz - 1 : z0 - 1;               // plane index being staged next
    auto stage = [&](int m) {
        const bool inpl = m >= 1 && m <= lzn;
        float *dst = raw + (m & 1) * C::RAW_BUF;
        const int base = kst * plane;
#pragma unroll
        for (int v = 0; v < 4; v++) cp_async16(dst + v * C::RAW_FIELD + my, src[v] + base + rowoff + i);
        if (inpl) {
            if (bot || top) {
#pragma unroll
                for (int v = 0; v < 4; v++) cp_async16(dst + v * C::RAW_FIELD + myh, src[v] + base + hrowoff + i);
            }
            if (edge_l) {
#pragma unroll
                for (int v = 0; v < 4; v++)
                    cp_async4(dst + v * C::RAW_FIELD + (row + 1) * C::RS + 3, src[v] + base + rowoff + im);
            }
            if (edge_r) {
#pragma unroll
                for (int v = 0; v < 4; v++)
                    cp_async4(dst + v * C::RAW_FIELD + (row + 1) * C::RS + 132, src[v] + base + rowoff + ip);
            }
        }
        cp_async_commit();
        kst = kst + 1 == g.nz ? 0 : kst + 1;
    };

    const f2 zero = splat(0.0f);
    Quad pend, zup;          // plane m-1 awaiting its +z term; h*(U + F_z) of plane m-1
#pragma unroll
    for (int p = 0; p < 2; p++)
#pragma unroll
        for (int v = 0; v < 4; v++) { pend.v[p][v] = zero; zup.v[p][v] = zero; }

    int oprev = 0;           // flat index of this thread's quad in plane m-1
    int ocur = (z0 == 0 ? g.nz - 1 : z0 - 1) * plane + rowoff + i;
    int kcur = z0 == 0 ? g.nz - 1 : z0 - 1;

    stage(0);
    for (int m = 0; m <= lzn + 1; m++) {
        cp_async_wait_all();                            // this thread's part of plane m has landed
        if (m + 1 <= lzn + 1) stage(m + 1);
        const bool inpl = m >= 1 && m <= lzn;
        const bool fin = m >= 2;
        const float *buf = raw + (m & 1) * C::RAW_BUF;
        float *wp = wy + (m & 1) * C::W_BUF;             // [0]: plus slots, [1]: minus slots
        float *wm = wp + 4 * C::W_COMP;
        const unsigned bar = bar0 + 8 * (m & 1);

        // early loads for the chemistry of plane m-1
        float4 x4 = make_float4(0.f, 0.f, 0.f, 0.f), T4 = x4, h4 = make_float4(1.f, 1.f, 1.f, 1.f);
        bool has_src = false;
        if (fin) {
            x4 = *reinterpret_cast<const float4 *>(f.x + oprev);
            T4 = *reinterpret_cast<const float4 *>(f.T + oprev);
            h4 = __ldg(reinterpret_cast<const float4 *>(f.nH + oprev));
            has_src = source_segment_flag(f, oprev);
        }

        // ---- closure of the staged row
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
        // ---- y: publish (U + F_y) for the row above, (U - F_y) for the row below; then arrive
        if (inpl) {
            {
                f2 F[2][4];
                flux_row(1, u.v[0], a[0], s[0], F[0]);
                flux_row(1, u.v[1], a[1], s[1], F[1]);
#pragma unroll
                for (int v = 0; v < 4; v++) {
                    if (!top) {
                        const f2 w0 = u.v[0][v] + F[0][v], w1 = u.v[1][v] + F[1][v];
                        *reinterpret_cast<float4 *>(wp + v * C::W_COMP + (row + 1) * 128 + 4 * lane) =
                            make_float4(lo(w0), hi(w0), lo(w1), hi(w1));
                    }
                    if (!bot) {
                        const f2 w0 = u.v[0][v] - F[0][v], w1 = u.v[1][v] - F[1][v];
                        *reinterpret_cast<float4 *>(wm + v * C::W_COMP + (row - 1) * 128 + 4 * lane) =
                            make_float4(lo(w0), hi(w0), lo(w1), hi(w1));
                    }
                }
            }
            if (bot || top) {       // the tile's y halo row: closure + F_y only (warp-uniform branch)
                const float4 n4 = *reinterpret_cast<const float4 *>(buf + myh);
                const float4 gx4 = *reinterpret_cast<const float4 *>(buf + C::RAW_FIELD + myh);
                const float4 gy4 = *reinterpret_cast<const float4 *>(buf + 2 * C::RAW_FIELD + myh);
                const float4 gz4 = *reinterpret_cast<const float4 *>(buf + 3 * C::RAW_FIELD + myh);
                f2 w[2][4];
#pragma unroll
                for (int p = 0; p < 2; p++) {
                    f2 e[4] = {ld_pair(n4, p), ld_pair(gx4, p), ld_pair(gy4, p), ld_pair(gz4, p)};
                    f2 ea, es, F[4];
                    closure2(e[0], e[1], e[2], e[3], ea, es);
                    flux_row(1, e, ea, es, F);
#pragma unroll
                    for (int v = 0; v < 4; v++) w[p][v] = bot ? e[v] + F[v] : e[v] - F[v];
                }
                float *wdst = bot ? wp : wm + (TY - 1) * 128;
#pragma unroll
                for (int v = 0; v < 4; v++)
                    *reinterpret_cast<float4 *>(wdst + v * C::W_COMP + 4 * lane) =
                        make_float4(lo(w[0][v]), hi(w[0][v]), lo(w[1][v]), hi(w[1][v]));
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar);
        }
        // ---- z: complete plane m-1, start plane m, seed plane m+1
        Quad t;
#pragma unroll
        for (int p = 0; p < 2; p++) {
            f2 F[4];
            flux_row(2, u.v[p], a[p], s[p], F);
#pragma unroll
            for (int v = 0; v < 4; v++) {
                pend.v[p][v] = fma2(u.v[p][v] - F[v], c.h, pend.v[p][v]);
                t.v[p][v] = fma2(u.v[p][v], c.keep, zup.v[p][v]);
                zup.v[p][v] = (u.v[p][v] + F[v]) * c.h;
            }
        }
        // ---- x: (U + F_x) of the cell to the left, (U - F_x) of the cell to the right
        if (inpl) {
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
                const int cl = (row + 1) * C::RS + 3, cr = (row + 1) * C::RS + 132;
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
                const f2 sx0 = pk(left + hi(Wm[0][v]), lo(Wp[0][v]) + lo(Wm[1][v]));
                const f2 sx1 = pk(hi(Wp[0][v]) + hi(Wm[1][v]), lo(Wp[1][v]) + right);
                t.v[0][v] = fma2(sx0, c.h, t.v[0][v]);
                t.v[1][v] = fma2(sx1, c.h, t.v[1][v]);
            }
        }
        // ---- plane m-1 has all six contributions: inject, one chemistry sub-step, store
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
        // ---- y terms of plane m (every warp arrived long ago), written straight into the carried registers
        if (inpl) {
            mbar_wait(bar, ((m - 1) >> 1) & 1);
            const int rp = row * 128 + 4 * lane;
#pragma unroll
            for (int v = 0; v < 4; v++) {
                const float4 yp = *reinterpret_cast<const float4 *>(wp + v * C::W_COMP + rp);
                const float4 ym = *reinterpret_cast<const float4 *>(wm + v * C::W_COMP + rp);
#pragma unroll
                for (int p = 0; p < 2; p++)
                    pend.v[p][v] = fma2(ld_pair(yp, p) + ld_pair(ym, p), c.h, t.v[p][v]);
            }
        } else {
            pend = t;
        }
        oprev = ocur;
        kcur = kcur + 1 == g.nz ? 0 : kcur + 1;
        ocur = kcur * plane + rowoff + i;
    }
}

inline bool v3_grid_ok(const Grid &g, int ty) { return g.nx % 128 == 0 && ty >= 2 && g.ny % ty == 0; }
inline bool v3_shape_ok(int tile_y, int tile_z) {
    return (tile_y == 0 || tile_y == 4 || tile_y == 8 || tile_y == 16) && tile_z >= 0;
}
inline int v3_pick_ty(const Grid &g, int tile_y) {
    if (tile_y > 0) return v3_grid_ok(g, tile_y) ? tile_y : 0;
    if (v3_grid_ok(g, 8)) return 8;
    if (v3_grid_ok(g, 4)) return 4;
    return 0;
}

inline int v3_default_lz(const Grid &g, int ty, int tile_z) {
    if (tile_z > 0) return tile_z < g.nz ? tile_z : g.nz;
    const long tiles_xy = (long)(g.nx / 128) * (g.ny / ty);
    int lz = 64;      // largest power of two <= 64 that still gives >= 4 CTAs per SM
    while (lz > 4 && tiles_xy * ((g.nz + lz - 1) / lz) < 4L * 148) lz >>= 1;
    return lz < g.nz ? lz : g.nz;
}

template <int FLAGS, int TY>
cudaError_t launch_step_v3_ty(const FieldsIO &f, const Grid &g, const StepConst &c, int tile_z, cudaStream_t stream) {
    using C = V3Cfg<TY>;
    static bool attr_done = false;     // one per instantiation
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(step_v3_kernel<FLAGS, TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    const int lz = v3_default_lz(g, TY, tile_z);
    const dim3 grid(g.nx / 128, g.ny / TY, (g.nz + lz - 1) / lz);
    step_v3_kernel<FLAGS, TY><<<grid, C::THREADS, C::SMEM, stream>>>(f, g, c, lz);
    return cudaGetLastError();
}

// ty must come from v3_pick_ty (non-zero)
template <int FLAGS>
cudaError_t launch_step_v3(const FieldsIO &f, const Grid &g, const StepConst &c, int ty, int tile_z, cudaStream_t stream) {
    if (ty == 4) return launch_step_v3_ty<FLAGS, 4>(f, g, c, tile_z, stream);
    if (ty == 16) return launch_step_v3_ty<FLAGS, 16>(f, g, c, tile_z, stream);
    return launch_step_v3_ty<FLAGS, 8>(f, g, c, tile_z, stream);
}

}  // namespace aton
