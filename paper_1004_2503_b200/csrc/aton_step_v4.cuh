// Fused step kernel, variant 4 (the product kernel for grids with nx % 32 == 0 and ny % 4 == 0, or nx % 64 == 0
// and ny % 2 == 0; the comments below describe the default 32 x 4 tile, WXQ = 8):
// WARP-AUTONOMOUS tiles.  Transport + one chemistry sub-step in one pass over HBM (52 B per cell-update);
// source cells and cells that need sub-cycling are queued per warp and redone in batches (v4_fix_batch).
//
// Why: profiles/r01_c_step_v3_512.md -- with CTA-wide tiles every warp spent 20 % of its time spinning on the
// per-plane CTA barrier (the slowest of 8 warps, its DRAM latency hiccups and the two edge warps' extra
// halo row set the pace), 9 % on the source-mask load and 3 % in source binary searches, at 4 warps per
// scheduler with nothing else to issue.  Here no warp ever waits for another warp:
//  * a warp owns a tile of 32 x-cells x 4 rows (lane = row r = lane>>3, quad q = lane&7) and marches
//    through a z-chunk; x neighbours come from shuffles inside the row's 8 lanes, y neighbours through a
//    4 KB warp-private shared-memory patch fenced by __syncwarp, z neighbours stay in registers;
//  * the tile's own halo (the rows below / above, the cells left / right) is staged and closed by the warp
//    itself in one extra pass (lanes of rows 0 and 3 take the y halo rows, lanes q = 0 / 7 the x halo
//    cells): ~10 % more instructions and 1.6x more L2->SM traffic on (N, G) for zero synchronisation;
//    HBM traffic is unchanged (the re-reads hit L2: neighbouring tiles run at the same time);
//  * the z loop is peeled (first two / last iteration) so the steady-state body is one straight-line
//    block: no `if (in plane)`, `if (finished)`, no divergent halo branches (predicated stores instead),
//    no source lookups -- the scheduler interleaves the chemistry's MUFU chains with the transport FMAs;
//  * per-cell source flags come from a 1-bit-per-cell mask: a source cell is treated like a cell that
//    needs sub-cycling (chemistry result discarded, flagged); the fix-up kernel injects and sub-cycles.
//  * cells that need sub-cycling (and the source cells) keep their transported values, are flagged in a 1-bit-per-cell
//    mask and are redone by step_fixup_kernel (aton_fixup.cuh).  Redoing them inside this kernel (a warp-private queue
//    drained 32 cells at a time) was built and measured in round 2: slower in every state (profiles/r02_b_fixup.md).
#pragma once
#include <type_traits>

#include "aton_fixup.cuh"
#include "aton_step_fused.cuh"

namespace aton {

#ifndef ATON_V4_WARPS
#define ATON_V4_WARPS 4
#endif
// WXQ = quads per tile row: 8 -> a 32 x 4 tile (the default), 16 -> 64 x 2
template <int WXQ>
struct V4Cfg {
    static constexpr int WX = 4 * WXQ, WY = 32 / WXQ;    // cells per warp tile
    static constexpr int RS = WX + 8;                    // raw row: quads at col 4 + 4q, x halos at 3 and 4 + WX
    static constexpr int RAW_FIELD = (WY + 2) * RS;      // row slots 0 / WY+1 = y halo rows
    static constexpr int RAW_BUF = 4 * RAW_FIELD;        // [field][slot][RS]
    static constexpr int W_COMP = WY * WX;               // plus: slot r = (U+F_y) of row r-1; minus: slot r = row r+1
    static constexpr int W_SIGN = 4 * W_COMP;            // [comp][slot][WX]
    static constexpr int WARP_FLOATS = 2 * RAW_BUF + 2 * W_SIGN;
    static constexpr int WARPS = ATON_V4_WARPS, THREADS = 32 * WARPS;
    // 47 104 B per CTA for the 32 x 4 tile: 4 CTAs fit the 196 KB shared-memory carve-out and leave 60 KB of L1 for the
    // halo re-reads.  768 B more per warp (tried: a queue of deferred cells) falls into the 228 KB carve-out, 28 KB of
    // L1, and costs 3.4 ms per 1024^3 step (profiles/r02_b_fixup.md).
    static constexpr size_t SMEM = (size_t)WARPS * WARP_FLOATS * sizeof(float);
};

#ifndef ATON_V4_X
#define ATON_V4_X 7      // codegen choices (measured: profiles/r01_d_step_v4.md); bits: 1 edge selects by slct; 2 predicated y stores; 4 predicated staging
#endif
// d = (c >= 0) ? a : b in one instruction
__device__ __forceinline__ float slct(float a, float b, int c) {
    float d;
    asm("slct.f32.s32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "r"(c));
    return d;
}
__device__ __forceinline__ void sts128_if(float *p, float a, float b, float c, float d, int pred) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.s32 p, %5, 0;\n@p st.shared.v4.f32 [%0], {%1, %2, %3, %4};\n}"
                 ::"r"(smem_u32(p)), "f"(a), "f"(b), "f"(c), "f"(d), "r"(pred) : "memory");
}
#ifndef ATON_V4_CS
#define ATON_V4_CS 0     // bit 0: streaming loads of x, T, n_H; bit 1: streaming stores
#endif
#ifndef ATON_V4_CA
#define ATON_V4_CA 1     // 1: stage quads through L1 (cp.async.ca) so that a neighbour tile's halo request can hit there
#endif
__device__ __forceinline__ void cp_async16_own(void *smem, const void *gmem) {
#if ATON_V4_CA
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
#else
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
#endif
}
__device__ __forceinline__ void cp_async16_if(void *smem, const void *gmem, int pred) {
#if ATON_V4_CA
    asm volatile("{\n.reg .pred p;\nsetp.ne.s32 p, %2, 0;\n@p cp.async.ca.shared.global [%0], [%1], 16;\n}"
                 ::"r"(smem_u32(smem)), "l"(gmem), "r"(pred) : "memory");
    return;
#endif
    asm volatile("{\n.reg .pred p;\nsetp.ne.s32 p, %2, 0;\n@p cp.async.cg.shared.global [%0], [%1], 16;\n}"
                 ::"r"(smem_u32(smem)), "l"(gmem), "r"(pred) : "memory");
}
__device__ __forceinline__ void cp_async4_if(void *smem, const void *gmem, int pred) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.s32 p, %2, 0;\n@p cp.async.ca.shared.global [%0], [%1], 4;\n}"
                 ::"r"(smem_u32(smem)), "l"(gmem), "r"(pred) : "memory");
}
// x, T, n_H, source bits of the plane being finished staged by cp.async through the slots of the plane just read: no
// register is held while they travel.  Pays in variant 5 (12.98 -> 12.4 ms per 1024^3 launch), not here (13.2 -> 13.45 ms:
// the extra LDGSTS compete with the halo re-reads for this kernel's L1): profiles/r02_d_step_v5.md
#ifndef ATON_V4_XT
#define ATON_V4_XT 0
#endif
#ifndef ATON_V5_XT
#define ATON_V5_XT 1
#endif
#ifndef ATON_PF
#define ATON_PF 1        // L2 prefetch of x, T, n_H, source bits two planes ahead: 1 per thread (prefetch.global.L2), 2 bulk per row
#endif
#ifndef ATON_V4_MINB
#define ATON_V4_MINB 4
#endif
template <int FLAGS, int WXQ>
__global__ void __launch_bounds__(V4Cfg<WXQ>::THREADS, ATON_V4_MINB)
step_v4_kernel(FieldsIO f, Grid g, StepConst c, int lz, int zb, int ze) {
    using C = V4Cfg<WXQ>;
    extern __shared__ __align__(16) float smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int r = lane / WXQ, q = lane % WXQ;
    const int xt = blockIdx.x * C::WARPS + warp;         // x tile of this warp
    if (xt * C::WX >= g.nx) return;                      // ragged last CTA in x: warps are independent
    float *raw = smem + warp * C::WARP_FLOATS;           // [2][4][6][RS], thread-private entries
    float *wyp = raw + 2 * C::RAW_BUF;                   // [4][4][32] plus terms
    float *wym = wyp + C::W_SIGN;                        //            minus terms

    // planes [zb, ze) are advanced: the whole periodic grid (0, nz), or a slab's own planes (1, nz - 1) whose
    // ghost planes 0 and nz - 1 hold the neighbours' boundary planes (no wrap is ever taken then)
    const int x0 = xt * C::WX, y0 = blockIdx.y * C::WY, z0 = zb + blockIdx.z * lz;
    const int lzn = min(lz, ze - z0);
    const int plane = g.nx * g.ny;
    const int rowoff = (y0 + r) * g.nx + x0 + 4 * q;     // own quad inside a plane
    // y halo row of this lane: rows 0 / 3 take the row below / above the tile (others: a harmless re-read)
    const bool hbot = r == 0, htop = r == C::WY - 1;
    const int jh = hbot ? (y0 == 0 ? g.ny - 1 : y0 - 1) : (htop ? (y0 + C::WY == g.ny ? 0 : y0 + C::WY) : y0 + r);
    const int hoff = jh * g.nx + x0 + 4 * q;
    const int hslot = hbot ? 0 : (htop ? C::WY + 1 : r + 1);
    // x halo cell of this lane: q = 0 the cell left of the tile, q = 7 the cell right of it
    const bool edge_l = q == 0, edge_r = q == WXQ - 1;
    const int xh = edge_l ? (x0 == 0 ? g.nx - 1 : x0 - 1) : (x0 + C::WX == g.nx ? 0 : x0 + C::WX);
    const int xoff = (y0 + r) * g.nx + xh;
    const int my = (r + 1) * C::RS + 4 + 4 * q;          // own quad inside a raw field
    const int myh = hslot * C::RS + 4 + 4 * q;           // halo-row quad
    const int mxh = (r + 1) * C::RS + (edge_l ? 3 : 4 + C::WX); // x halo cell (valid for edge lanes)
    const float *src[4] = {f.N, f.Gx, f.Gy, f.Gz};

    int kst = z0 == 0 ? g.nz - 1 : z0 - 1;               // plane index staged next (periodic)
    auto stage = [&](int m, bool inpl) {
        float *dst = raw + (m & 1) * C::RAW_BUF;
        const int base = kst * plane;
#pragma unroll
        for (int v = 0; v < 4; v++) cp_async16_own(dst + v * C::RAW_FIELD + my, src[v] + base + rowoff);
        if (inpl) {
#if ATON_V4_X & 4
#pragma unroll
            for (int v = 0; v < 4; v++) cp_async16_if(dst + v * C::RAW_FIELD + myh, src[v] + base + hoff, hbot || htop);
#pragma unroll
            for (int v = 0; v < 4; v++) cp_async4_if(dst + v * C::RAW_FIELD + mxh, src[v] + base + xoff, edge_l || edge_r);
#else
            if (hbot || htop) {
#pragma unroll
                for (int v = 0; v < 4; v++) cp_async16(dst + v * C::RAW_FIELD + myh, src[v] + base + hoff);
            }
            if (edge_l || edge_r) {
#pragma unroll
                for (int v = 0; v < 4; v++) cp_async4(dst + v * C::RAW_FIELD + mxh, src[v] + base + xoff);
            }
#endif
        }
#if ATON_PF == 1
        if (inpl) {      // the plane is finished two iterations from now: its x, T, n_H and source bits wait in L2 by then
            prefetch_l2(f.x + base + rowoff);
            prefetch_l2(f.T + base + rowoff);
            prefetch_l2(f.nH + base + rowoff);
            if (q == 0) prefetch_l2(f.src_bits + ((unsigned)(base + rowoff) >> 5));
        }
#elif ATON_PF == 2
        if (inpl && q == 0) {
            prefetch_l2_bulk(f.x + base + rowoff, 4 * C::WX);
            prefetch_l2_bulk(f.T + base + rowoff, 4 * C::WX);
            prefetch_l2_bulk(f.nH + base + rowoff, 4 * C::WX);
            prefetch_l2(f.src_bits + ((unsigned)(base + rowoff) >> 5));
        }
#endif
        cp_async_commit();
        kst = kst + 1 == g.nz ? 0 : kst + 1;
    };

    const f2 zero = splat(0.0f);
    Quad pend, zup;          // plane m-1 awaiting its +z term; h*(U + F_z) of plane m-1
#pragma unroll
    for (int p = 0; p < 2; p++)
#pragma unroll
        for (int v = 0; v < 4; v++) { pend.v[p][v] = zero; zup.v[p][v] = zero; }

    int kcur = z0 == 0 ? g.nz - 1 : z0 - 1;
    int ocur = kcur * plane + rowoff;    // flat index of this thread's quad in plane m
    int oprev = 0;                       //                                  in plane m-1
    int m = 0;

    // one z iteration; INPL: plane m belongs to the chunk (x / y terms needed); FIN: plane m-1 is finished here
    auto iter = [&](auto inpl_tag, auto fin_tag, bool stage_next, bool next_inpl) {
        constexpr bool INPL = decltype(inpl_tag)::value, FIN = decltype(fin_tag)::value;
        cp_async_wait_all();                             // this thread's part of plane m has landed
        float *buf = raw + (m & 1) * C::RAW_BUF;
        // the staged quad of plane m goes to registers first: its slots are reused right away
        const float4 n4 = *reinterpret_cast<const float4 *>(buf + my);
        const float4 gx4 = *reinterpret_cast<const float4 *>(buf + C::RAW_FIELD + my);
        const float4 gy4 = *reinterpret_cast<const float4 *>(buf + 2 * C::RAW_FIELD + my);
        const float4 gz4 = *reinterpret_cast<const float4 *>(buf + 3 * C::RAW_FIELD + my);
#if ATON_V4_XT
        // x, T, n_H and the source bits of plane m-1 (finished at the end of this iteration) travel through the slots
        // just read: no register is held while they are on their way (profiles/r02_d_step_v5.md).  (The lanes of the
        // middle rows re-read their own slot in the halo pass below: whatever they find there is never stored.)
        if (FIN) {
            cp_async16(buf + my, f.x + oprev);
            cp_async16(buf + C::RAW_FIELD + my, f.T + oprev);
            cp_async16(buf + 2 * C::RAW_FIELD + my, f.nH + oprev);
            cp_async4(buf + 3 * C::RAW_FIELD + my, f.src_bits + ((unsigned)oprev >> 5));
            cp_async_commit();
        }
#endif
        if (stage_next) stage(m + 1, next_inpl);

#if !ATON_V4_XT
        // early loads for the chemistry of plane m-1
        float4 x4 = make_float4(0.f, 0.f, 0.f, 0.f), T4 = x4, h4 = make_float4(1.f, 1.f, 1.f, 1.f);
        unsigned srcw = 0;
        if (FIN) {
            x4 = *reinterpret_cast<const float4 *>(f.x + oprev);
            T4 = *reinterpret_cast<const float4 *>(f.T + oprev);
            h4 = __ldg(reinterpret_cast<const float4 *>(f.nH + oprev));
            srcw = __ldg(f.src_bits + ((unsigned)oprev >> 5));
        }
#endif
        // ---- closure of the staged quad
        Quad u;
        f2 a[2], s[2];
        {
#pragma unroll
            for (int p = 0; p < 2; p++) {
                u.v[p][0] = ld_pair(n4, p); u.v[p][1] = ld_pair(gx4, p);
                u.v[p][2] = ld_pair(gy4, p); u.v[p][3] = ld_pair(gz4, p);
                closure2(u.v[p][0], u.v[p][1], u.v[p][2], u.v[p][3], a[p], s[p]);
            }
        }
        Quad t;
        if (INPL) {
            __syncwarp();                                // every lane has consumed the previous plane's y terms
            // ---- y: publish (U + F_y) for the row above, (U - F_y) for the row below
            {
                f2 F[2][4];
                flux_row(1, u.v[0], a[0], s[0], F[0]);
                flux_row(1, u.v[1], a[1], s[1], F[1]);
#pragma unroll
                for (int v = 0; v < 4; v++) {
                    const f2 p0 = u.v[0][v] + F[0][v], p1 = u.v[1][v] + F[1][v];
                    const f2 m0 = u.v[0][v] - F[0][v], m1 = u.v[1][v] - F[1][v];
#if ATON_V4_X & 2
                    sts128_if(wyp + v * C::W_COMP + (r + 1) * C::WX + 4 * q, lo(p0), hi(p0), lo(p1), hi(p1), !htop);
                    sts128_if(wym + v * C::W_COMP + (r - 1) * C::WX + 4 * q, lo(m0), hi(m0), lo(m1), hi(m1), !hbot);
#else
                    if (!htop)
                        *reinterpret_cast<float4 *>(wyp + v * C::W_COMP + (r + 1) * C::WX + 4 * q) =
                            make_float4(lo(p0), hi(p0), lo(p1), hi(p1));
                    if (!hbot)
                        *reinterpret_cast<float4 *>(wym + v * C::W_COMP + (r - 1) * C::WX + 4 * q) =
                            make_float4(lo(m0), hi(m0), lo(m1), hi(m1));
#endif
                }
            }
            // ---- the tile's y halo rows (lanes of rows 0 and 3; the others compute and store nothing new)
            {
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
                    const f2 sg = splat(hbot ? 1.0f : -1.0f);
#pragma unroll
                    for (int v = 0; v < 4; v++) w[p][v] = fma2(F[v], sg, e[v]);
                }
                float *wdst = hbot ? wyp + 4 * q : wym + (C::WY - 1) * C::WX + 4 * q;
#if ATON_V4_X & 2
#pragma unroll
                for (int v = 0; v < 4; v++)
                    sts128_if(wdst + v * C::W_COMP, lo(w[0][v]), hi(w[0][v]), lo(w[1][v]), hi(w[1][v]), hbot || htop);
#else
                if (hbot || htop) {
#pragma unroll
                    for (int v = 0; v < 4; v++)
                        *reinterpret_cast<float4 *>(wdst + v * C::W_COMP) =
                            make_float4(lo(w[0][v]), hi(w[0][v]), lo(w[1][v]), hi(w[1][v]));
                }
#endif
            }
            __syncwarp();                                // y terms of the plane are visible to the warp
        }
        // ---- z: complete plane m-1, start plane m, seed plane m+1
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
        if (INPL) {
            f2 Wp[2][4], Wm[2][4];
#pragma unroll
            for (int p = 0; p < 2; p++) {
                f2 F[4];
                flux_row(0, u.v[p], a[p], s[p], F);
#pragma unroll
                for (int v = 0; v < 4; v++) { Wp[p][v] = u.v[p][v] + F[v]; Wm[p][v] = u.v[p][v] - F[v]; }
            }
            float xw[4];
            {   // the x halo cell of the edge lanes (all lanes run it; only q = 0 / WXQ - 1 use the result): (U + F_x) of
                // the cell left of the tile for q = 0, (U - F_x) of the cell right of it for q = WXQ - 1
                float e[4], ea, es;
#pragma unroll
                for (int v = 0; v < 4; v++) e[v] = buf[v * C::RAW_FIELD + mxh];
                closure1(e[0], e[1], e[2], e[3], ea, es);
                xterm1(e, ea, es, edge_r ? -1.0f : 1.0f, xw);
            }
#pragma unroll
            for (int v = 0; v < 4; v++) {
                float left = __shfl_up_sync(0xffffffffu, hi(Wp[1][v]), 1);
                float right = __shfl_down_sync(0xffffffffu, lo(Wm[0][v]), 1);
#if ATON_V4_X & 1
                left = slct(left, xw[v], q - 1);              // q == 0: the halo cell
                right = slct(right, xw[v], WXQ - 2 - q);      // q == WXQ - 1: the halo cell
#else
                left = edge_l ? xw[v] : left;
                right = edge_r ? xw[v] : right;
#endif
                const f2 sx0 = pk(left + hi(Wm[0][v]), lo(Wp[0][v]) + lo(Wm[1][v]));
                const f2 sx1 = pk(hi(Wp[0][v]) + hi(Wm[1][v]), lo(Wp[1][v]) + right);
                t.v[0][v] = fma2(sx0, c.h, t.v[0][v]);
                t.v[1][v] = fma2(sx1, c.h, t.v[1][v]);
            }
        }
        // ---- plane m-1 has all six contributions: one chemistry sub-step, store; source cells and cells
        //      that need sub-cycling keep their transported (N, G), old (x, T) and are flagged
        if (FIN) {
#if ATON_V4_XT
            if (stage_next) cp_async_wait_1(); else cp_async_wait_all();     // the next plane's staging may still fly
            const float4 x4 = *reinterpret_cast<const float4 *>(buf + my);
            const float4 T4 = *reinterpret_cast<const float4 *>(buf + C::RAW_FIELD + my);
            const float4 h4 = *reinterpret_cast<const float4 *>(buf + 2 * C::RAW_FIELD + my);
            const unsigned srcw = *reinterpret_cast<const unsigned *>(buf + 3 * C::RAW_FIELD + my);
#endif
            const unsigned srcn = (srcw >> (oprev & 31)) & 0xFu;
            f2 xs[2] = {pk(x4.x, x4.y), pk(x4.z, x4.w)}, Ts[2] = {pk(T4.x, T4.y), pk(T4.z, T4.w)};
            const f2 hs[2] = {pk(h4.x, h4.y), pk(h4.z, h4.w)};
            unsigned nib = 0;
#pragma unroll
            for (int p = 0; p < 2; p++)
                nib |= chem_fast2<FLAGS>(pend.v[p][0], pend.v[p][1], pend.v[p][2], pend.v[p][3], xs[p], Ts[p], hs[p], c,
                                         (srcn >> (2 * p)) & 3u)
                       << (2 * p);
#if ATON_V4_CS & 2       // written once, not read again this step: streaming stores
#define ATON_ST4(ptr, A, B) __stcs(reinterpret_cast<float4 *>(ptr + oprev), make_float4(lo(A), hi(A), lo(B), hi(B)))
#else
#define ATON_ST4(ptr, A, B) *reinterpret_cast<float4 *>(ptr + oprev) = make_float4(lo(A), hi(A), lo(B), hi(B))
#endif
            ATON_ST4(f.N1, pend.v[0][0], pend.v[1][0]);
            ATON_ST4(f.Gx1, pend.v[0][1], pend.v[1][1]);
            ATON_ST4(f.Gy1, pend.v[0][2], pend.v[1][2]);
            ATON_ST4(f.Gz1, pend.v[0][3], pend.v[1][3]);
            ATON_ST4(f.x, xs[0], xs[1]);
            ATON_ST4(f.T, Ts[0], Ts[1]);
#undef ATON_ST4
            if (nib) atomicOr(f.defer_mask + ((unsigned)oprev >> 5), nib << (oprev & 31));
        }
        // ---- y terms of plane m, written straight into the carried registers
        if (INPL) {
            const int rp = r * C::WX + 4 * q;
#pragma unroll
            for (int v = 0; v < 4; v++) {
                const float4 yp = *reinterpret_cast<const float4 *>(wyp + v * C::W_COMP + rp);
                const float4 ym = *reinterpret_cast<const float4 *>(wym + v * C::W_COMP + rp);
#pragma unroll
                for (int p = 0; p < 2; p++)
                    pend.v[p][v] = fma2(ld_pair(yp, p) + ld_pair(ym, p), c.h, t.v[p][v]);
            }
        } else {
            pend = t;
        }
        oprev = ocur;
        kcur = kcur + 1 == g.nz ? 0 : kcur + 1;
        ocur = kcur * plane + rowoff;
        m++;
    };

    const std::true_type yes{};
    const std::false_type no{};
    stage(0, false);
    iter(no, no, true, true);                  // m = 0: z halo plane below the chunk
    iter(yes, no, true, true);                 // m = 1: first own plane, nothing to finish yet
    while (m <= lzn) iter(yes, yes, true, true);   // steady state (the last one stages the z halo plane above)
    iter(no, yes, false, false);               // m = lzn + 1: z halo plane above, finishes plane lzn
}

// tile shapes: 32 x 4 (nx % 32 == 0, ny % 4 == 0; the default: 13.8 ms per 1024^3 step) or 64 x 2 (nx % 64 == 0,
// ny % 2 == 0; 14.1 ms: its 256-byte row segments stream better in isolation, but every row is then read twice
// and the tile halo costs more than the segments gain -- profiles/r01_e_tile_shape.md).  `tile_y` = 4 / 2 forces
// one, 0 picks 32 x 4 when the grid allows it.  Results do not depend on the shape (bitwise).  Returns WXQ or 0.
inline int v4_pick_wxq(const Grid &g, int tile_y) {
    const bool ok16 = g.nx % 64 == 0 && g.ny % 2 == 0, ok8 = g.nx % 32 == 0 && g.ny % 4 == 0;
    if (tile_y == 2) return ok16 ? 16 : 0;
    if (tile_y == 4) return ok8 ? 8 : 0;
    return ok8 ? 8 : (ok16 ? 16 : 0);
}
inline bool v4_grid_ok(const Grid &g) { return v4_pick_wxq(g, 0) != 0; }
inline bool v4_shape_ok(int tile_y, int tile_z) { return (tile_y == 0 || tile_y == 2 || tile_y == 4) && tile_z >= 0; }

template <int WXQ>
inline int v4_default_lz(const Grid &g, int tile_z, int nzr) {
    using C = V4Cfg<WXQ>;
    if (tile_z > 0) return tile_z < nzr ? tile_z : nzr;
    const long tiles_xy = (long)((g.nx / C::WX + C::WARPS - 1) / C::WARPS) * (g.ny / C::WY);
    int lz = 64;      // largest power of two <= 64 that still gives >= 4 waves of 4 CTAs per SM
    while (lz > 4 && tiles_xy * ((nzr + lz - 1) / lz) < 16L * 148) lz >>= 1;
    return lz < nzr ? lz : nzr;
}

template <int FLAGS, int WXQ>
cudaError_t launch_step_v4_wxq(const FieldsIO &f, const Grid &g, const StepConst &c, int tile_z, cudaStream_t stream,
                               int zb, int ze) {
    using C = V4Cfg<WXQ>;
    // the attribute is per device, not per process: set it at every launch (a cheap driver call)
    cudaError_t e = cudaFuncSetAttribute(step_v4_kernel<FLAGS, WXQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    const int lz = v4_default_lz<WXQ>(g, tile_z, ze - zb);
    const dim3 grid((g.nx / C::WX + C::WARPS - 1) / C::WARPS, g.ny / C::WY, (ze - zb + lz - 1) / lz);
    step_v4_kernel<FLAGS, WXQ><<<grid, C::THREADS, C::SMEM, stream>>>(f, g, c, lz, zb, ze);
    return cudaGetLastError();
}

// wxq must come from v4_pick_wxq (non-zero); planes [zb, ze) are advanced
template <int FLAGS>
cudaError_t launch_step_v4(const FieldsIO &f, const Grid &g, const StepConst &c, int wxq, int tile_z, cudaStream_t stream,
                           int zb, int ze) {
    if (wxq == 8) return launch_step_v4_wxq<FLAGS, 8>(f, g, c, tile_z, stream, zb, ze);
    return launch_step_v4_wxq<FLAGS, 16>(f, g, c, tile_z, stream, zb, ze);
}

}  // namespace aton
