// Fused step kernel, variant 5 (the PRODUCT kernel for grids with nx % 128 == 0 and ny % 8 == 0): ROW-WIDE warps,
// CTA-shared y terms consumed one plane late.  Transport + one chemistry sub-step in one pass over HBM (52 B per cell-update).
//
// Why (profiles/r01_e_tile_shape.md, r02_c_step_v4.md, r02_d_step_v5.md): variant 4's warp-autonomous 32 x 4 tile pays twice
// for its independence.  (i) Every warp request is four 128-byte row segments, and a z-march made of those streams at 0.83 of
// the copy peak (10.4 ms per 1024^3 step against 8.7 ms for 256- or 512-byte segments).  (ii) Every warp closes its own
// tile halo: three extra closure + flux passes per plane on top of the two of its own cells (17 % of the kernel's MUFU
// work).  Here
//  * a warp owns ONE ROW SEGMENT of 128 cells (lane q = the quad of cells 4q .. 4q+3): every load, cp.async and store of
//    a warp is 512 contiguous bytes; x neighbours by shuffles across the whole warp, z neighbours in registers;
//  * a CTA is W warps stacked in y (W = 16: a 128 x 16 tile, one CTA per SM; W = 8 when ny % 16 != 0, two per SM).  Every
//    row publishes (U + F_y) and (U - F_y) of plane m to a CTA-shared patch (double buffered by plane parity) and picks up
//    its neighbours' terms ONE ITERATION LATER, when plane m-1 is completed anyway (its +z term arrives with plane m).  The
//    only inter-warp synchronisation is one mbarrier phase per plane, arrived on right after the publish and waited for at
//    the top of the NEXT iteration: a warp may run a whole iteration ahead of its slowest neighbour before it stalls
//    (variant 3 of round 1 synchronised inside the iteration and lost 20 % of its issue slots to the barrier); a warp that
//    has to wait sleeps between probes;
//  * the two y halo rows of the CTA tile are closed by ONE warp each, a duty that rotates with the plane index
//    (below: warp m mod W, above: warp (m + W/2) mod W): 2 / W extra passes per warp and plane instead of 2;
//  * NO PLAIN GLOBAL LOAD in the loop: (N, G) of plane m+1 are staged by cp.async one plane ahead into thread-private
//    double-buffered slots; as soon as the quad of plane m has been read into registers its four slots receive x, T, n_H and
//    the source word of plane m-1 (the plane this iteration finishes) by cp.async too, fetched from L2 where a prefetch put
//    them two planes earlier.  No register waits for memory: with plain loads ptxas sank them to within 17-270 instructions
//    of their first use and every warp spent 27 % of its time on that scoreboard (profiles/r02_d_step_v5.md);
//  * everything else is variant 4's: the peeled z loop, the x halo cell of the edge lanes, one straight-line chemistry
//    sub-step (chem_fast2), source cells and cells that sub-cycle flagged in the 1-bit mask for step_fixup_kernel.  The
//    additions reach the accumulators in variant 4's order: results are bit-identical to variant 4's.
#pragma once
#include "aton_step_v4.cuh"

namespace aton {

template <int W>
struct V5Cfg {
    static constexpr int WX = 128;                       // cells per row segment (one warp)
    static constexpr int RS = WX + 8;                    // raw row: quads at col 4 + 4q, x halo cells at 3 and 4 + WX
    static constexpr int RAW_BUF = 4 * RS;               // [field][RS]
    static constexpr int RAW_WARP = 2 * RAW_BUF;         // double buffered, private to the warp
    static constexpr int Y_COMP = W * WX;                // [row][WX]
    static constexpr int Y_SIGN = 4 * Y_COMP;            // [comp][row][WX]
    static constexpr int Y_PAR = 2 * Y_SIGN;             // plus terms (consumed by the row above), minus terms
    static constexpr int H_SIDE = 4 * WX;                // raw y halo row: [field][WX]
    static constexpr int H_PAR = 2 * H_SIDE;             // below, above
    static constexpr int THREADS = 32 * W;
    static constexpr int FLOATS = W * RAW_WARP + 2 * Y_PAR + 2 * H_PAR;
    static constexpr size_t SMEM = (size_t)FLOATS * sizeof(float) + 16;   // + the mbarrier
};

__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar) {
    asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.release.cta.shared::cta.b64 st, [%0];\n}" ::"r"(smem_u32(bar)) : "memory");
}
#ifndef ATON_V5_SLEEP_NS
#define ATON_V5_SLEEP_NS 64u    // back-off of a warp that is ahead of its CTA: it sleeps instead of spinning through issue slots
#endif
__device__ __forceinline__ bool mbar_test(unsigned long long *bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n.reg .pred p;\n"
        "mbarrier.try_wait.parity.acquire.cta.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    while (!mbar_test(bar, parity)) {
#if ATON_V5_SLEEP_NS > 0
        __nanosleep(ATON_V5_SLEEP_NS);
#endif
    }
}

template <int FLAGS, int W>
__global__ void __launch_bounds__(V5Cfg<W>::THREADS, 512 / V5Cfg<W>::THREADS)
step_v5_kernel(FieldsIO f, Grid g, StepConst c, int lz, int zb, int ze) {
    using C = V5Cfg<W>;
    extern __shared__ __align__(16) float smem[];
    const int q = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float *raw = smem + warp * C::RAW_WARP;              // [2][4][RS], thread-private entries
    float *ypat = smem + W * C::RAW_WARP;                // [2 parity][plus, minus][4][W][WX]
    float *hraw = ypat + 2 * C::Y_PAR;                   // [2 parity][below, above][4][WX]
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(hraw + 2 * C::H_PAR);
    if (threadIdx.x == 0) mbar_init(bar, W);
    __syncthreads();

    // planes [zb, ze) are advanced (the periodic grid, or a slab's own planes between its two ghost planes)
    const int x0 = blockIdx.x * C::WX, y0 = blockIdx.y * W, z0 = zb + blockIdx.z * lz;
    const int lzn = min(lz, ze - z0);
    const int plane = g.nx * g.ny;
    const int rowoff = (y0 + warp) * g.nx + x0 + 4 * q;  // own quad inside a plane
    // the tile's y halo rows (periodic)
    const int jb = y0 == 0 ? g.ny - 1 : y0 - 1, jt = y0 + W == g.ny ? 0 : y0 + W;
    const int hoff_b = jb * g.nx + x0 + 4 * q, hoff_t = jt * g.nx + x0 + 4 * q;
    // x halo cell of the edge lanes
    const bool edge_l = q == 0, edge_r = q == 31;
    const int xh = edge_l ? (x0 == 0 ? g.nx - 1 : x0 - 1) : (x0 + C::WX == g.nx ? 0 : x0 + C::WX);
    const int xoff = (y0 + warp) * g.nx + xh;
    const int my = 4 + 4 * q;                            // own quad inside a raw field
    const int mxh = edge_l ? 3 : 4 + C::WX;              // x halo cell (valid for edge lanes)
    const float *src[4] = {f.N, f.Gx, f.Gy, f.Gz};

    // halo duty of plane m: below-row for (m - warp) % W == 0, above-row for (m - warp) % W == W / 2
    auto duty_of = [&](int m) { return (m - warp) & (W - 1); };

    int kst = z0 == 0 ? g.nz - 1 : z0 - 1;               // plane index staged next (periodic)
    auto stage = [&](int m, bool inpl) {
        float *dst = raw + (m & 1) * C::RAW_BUF;
        const int base = kst * plane;
#pragma unroll
        for (int v = 0; v < 4; v++) cp_async16(dst + v * C::RS + my, src[v] + base + rowoff);
        if (inpl) {
#pragma unroll
            for (int v = 0; v < 4; v++) cp_async4_if(dst + v * C::RS + mxh, src[v] + base + xoff, edge_l || edge_r);
            const int d = duty_of(m);
            if (d == 0 || d == W / 2) {                  // warp-uniform
                float *hd = hraw + (m & 1) * C::H_PAR + (d ? C::H_SIDE : 0) + 4 * q;
                const int ho = base + (d ? hoff_t : hoff_b);
#pragma unroll
                for (int v = 0; v < 4; v++) cp_async16(hd + v * C::WX, src[v] + ho);
            }
        }
#if ATON_PF == 1
        if (inpl) {      // the plane is finished two iterations from now: its x, T, n_H and source bits wait in L2 by then
            prefetch_l2(f.x + base + rowoff);
            prefetch_l2(f.T + base + rowoff);
            prefetch_l2(f.nH + base + rowoff);
            if ((q & 7) == 0) prefetch_l2(f.src_bits + ((unsigned)(base + rowoff) >> 5));
        }
#elif ATON_PF == 2
        if (inpl && q == 0) {
            prefetch_l2_bulk(f.x + base + rowoff, 4 * C::WX);
            prefetch_l2_bulk(f.T + base + rowoff, 4 * C::WX);
            prefetch_l2_bulk(f.nH + base + rowoff, 4 * C::WX);
            prefetch_l2_bulk(f.src_bits + ((unsigned)(base + rowoff) >> 5), 16);
        }
#endif
        cp_async_commit();
        kst = kst + 1 == g.nz ? 0 : kst + 1;
    };

    const f2 zero = splat(0.0f);
    Quad pend, zup;          // plane m-1 awaiting its y and +z terms; h*(U + F_z) of plane m-1
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
        // every row has published plane m-1 (and with that has consumed plane m-2: the patch of parity m & 1 and the
        // halo staging of parity (m + 1) & 1 are free)
        if (FIN) mbar_wait(bar, (unsigned)(m & 1));
        float *buf = raw + (m & 1) * C::RAW_BUF;
        // the staged quad of plane m goes to registers first: its slots are reused right away
        const float4 n4 = *reinterpret_cast<const float4 *>(buf + my);
        const float4 gx4 = *reinterpret_cast<const float4 *>(buf + C::RS + my);
        const float4 gy4 = *reinterpret_cast<const float4 *>(buf + 2 * C::RS + my);
        const float4 gz4 = *reinterpret_cast<const float4 *>(buf + 3 * C::RS + my);
#if ATON_V5_XT
        // x, T, n_H and the source bits of plane m-1 (finished at the end of this iteration) travel through the slots
        // just read: no register is held while they are on their way (profiles/r02_d_step_v5.md)
        if (FIN) {
            cp_async16(buf + my, f.x + oprev);
            cp_async16(buf + C::RS + my, f.T + oprev);
            cp_async16(buf + 2 * C::RS + my, f.nH + oprev);
            cp_async4(buf + 3 * C::RS + my, f.src_bits + ((unsigned)oprev >> 5));
            cp_async_commit();
        }
#endif
        if (stage_next) stage(m + 1, next_inpl);

#if !ATON_V5_XT
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
        // ---- y terms of plane m-1 from the rows below and above (published one iteration ago)
        if (FIN) {
            const float *yp = ypat + ((m - 1) & 1) * C::Y_PAR + warp * C::WX + 4 * q, *ym = yp + C::Y_SIGN;
#pragma unroll
            for (int v = 0; v < 4; v++) {
                const float4 a4 = *reinterpret_cast<const float4 *>(yp + v * C::Y_COMP);
                const float4 b4 = *reinterpret_cast<const float4 *>(ym + v * C::Y_COMP);
#pragma unroll
                for (int p = 0; p < 2; p++)
                    pend.v[p][v] = fma2(ld_pair(a4, p) + ld_pair(b4, p), c.h, pend.v[p][v]);
            }
        }
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
            // ---- y: publish (U + F_y) for the row above, (U - F_y) for the row below
            float *yp = ypat + (m & 1) * C::Y_PAR + 4 * q, *ym = yp + C::Y_SIGN;
            {
                f2 F[2][4];
                flux_row(1, u.v[0], a[0], s[0], F[0]);
                flux_row(1, u.v[1], a[1], s[1], F[1]);
#pragma unroll
                for (int v = 0; v < 4; v++) {
                    const f2 p0 = u.v[0][v] + F[0][v], p1 = u.v[1][v] + F[1][v];
                    const f2 m0 = u.v[0][v] - F[0][v], m1 = u.v[1][v] - F[1][v];
                    sts128_if(yp + v * C::Y_COMP + (warp + 1) * C::WX, lo(p0), hi(p0), lo(p1), hi(p1), warp != W - 1);
                    sts128_if(ym + v * C::Y_COMP + (warp - 1) * C::WX, lo(m0), hi(m0), lo(m1), hi(m1), warp != 0);
                }
            }
            // ---- the tile's y halo rows: one warp each, the duty rotates with the plane
            const int d = duty_of(m);
            if (d == 0 || d == W / 2) {
                const float *hb = hraw + (m & 1) * C::H_PAR + (d ? C::H_SIDE : 0) + 4 * q;
                const float4 n4 = *reinterpret_cast<const float4 *>(hb);
                const float4 gx4 = *reinterpret_cast<const float4 *>(hb + C::WX);
                const float4 gy4 = *reinterpret_cast<const float4 *>(hb + 2 * C::WX);
                const float4 gz4 = *reinterpret_cast<const float4 *>(hb + 3 * C::WX);
                const f2 sg = splat(d ? -1.0f : 1.0f);
                f2 w[2][4];
#pragma unroll
                for (int p = 0; p < 2; p++) {
                    f2 e[4] = {ld_pair(n4, p), ld_pair(gx4, p), ld_pair(gy4, p), ld_pair(gz4, p)};
                    f2 ea, es, F[4];
                    closure2(e[0], e[1], e[2], e[3], ea, es);
                    flux_row(1, e, ea, es, F);
#pragma unroll
                    for (int v = 0; v < 4; v++) w[p][v] = fma2(F[v], sg, e[v]);
                }
                float *wdst = d ? ym + (W - 1) * C::WX : yp;      // above: minus terms for row W-1; below: plus for row 0
#pragma unroll
                for (int v = 0; v < 4; v++)
                    *reinterpret_cast<float4 *>(wdst + v * C::Y_COMP) =
                        make_float4(lo(w[0][v]), hi(w[0][v]), lo(w[1][v]), hi(w[1][v]));
            }
            __syncwarp();
            if (q == 0) mbar_arrive(bar);                // this row's terms of plane m are out
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
            {   // the x halo cell of the edge lanes (all lanes run it; only q = 0 / 31 use the result): (U + F_x) of the
                // cell left of the row for lane 0, (U - F_x) of the cell right of it for lane 31
                float e[4], ea, es;
#pragma unroll
                for (int v = 0; v < 4; v++) e[v] = buf[v * C::RS + mxh];
                closure1(e[0], e[1], e[2], e[3], ea, es);
                xterm1(e, ea, es, edge_r ? -1.0f : 1.0f, xw);
            }
#pragma unroll
            for (int v = 0; v < 4; v++) {
                float left = __shfl_up_sync(0xffffffffu, hi(Wp[1][v]), 1);
                float right = __shfl_down_sync(0xffffffffu, lo(Wm[0][v]), 1);
                left = slct(left, xw[v], q - 1);              // q == 0: the halo cell
                right = slct(right, xw[v], 30 - q);           // q == 31: the halo cell
                const f2 sx0 = pk(left + hi(Wm[0][v]), lo(Wp[0][v]) + lo(Wm[1][v]));
                const f2 sx1 = pk(hi(Wp[0][v]) + hi(Wm[1][v]), lo(Wp[1][v]) + right);
                t.v[0][v] = fma2(sx0, c.h, t.v[0][v]);
                t.v[1][v] = fma2(sx1, c.h, t.v[1][v]);
            }
        }
        // ---- plane m-1 has all six contributions: one chemistry sub-step, store; source cells and cells
        //      that need sub-cycling keep their transported (N, G), old (x, T) and are flagged
        if (FIN) {
#if ATON_V5_XT
            if (stage_next) cp_async_wait_1(); else cp_async_wait_all();     // the next plane's staging may still fly
            const float4 x4 = *reinterpret_cast<const float4 *>(buf + my);
            const float4 T4 = *reinterpret_cast<const float4 *>(buf + C::RS + my);
            const float4 h4 = *reinterpret_cast<const float4 *>(buf + 2 * C::RS + my);
            const unsigned srcw = *reinterpret_cast<const unsigned *>(buf + 3 * C::RS + my);
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
        pend = t;                        // plane m waits for its y terms (next iteration) and its +z term
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

// grids variant 5 tiles: nx % 128 == 0 and ny % W == 0 (W = 16 rows per CTA when ny allows it, else 8; tile_y forces one)
inline int v5_pick_w(const Grid &g, int tile_y) {
    if (g.nx % 128 != 0) return 0;
    if (tile_y == 16) return g.ny % 16 == 0 ? 16 : 0;
    if (tile_y == 8) return g.ny % 8 == 0 ? 8 : 0;
    if (tile_y == 0) return g.ny % 16 == 0 ? 16 : (g.ny % 8 == 0 ? 8 : 0);   // 16 rows: 12.17 against 12.35 ms at 1024^3
    return 0;
}
inline bool v5_shape_ok(int tile_y, int tile_z) { return (tile_y == 0 || tile_y == 8 || tile_y == 16) && tile_z >= 0; }

template <int W>
inline int v5_default_lz(const Grid &g, int tile_z, int nzr) {
    if (tile_z > 0) return tile_z < nzr ? tile_z : nzr;
    const long tiles_xy = (long)(g.nx / 128) * (g.ny / W);
    const long per_wave = 148L * (512 / (32 * W));
    int lz = 128;     // largest power of two <= 128 that still gives >= 4 waves
    while (lz > 4 && tiles_xy * ((nzr + lz - 1) / lz) < 4 * per_wave) lz >>= 1;
    return lz < nzr ? lz : nzr;
}

template <int FLAGS, int W>
cudaError_t launch_step_v5_w(const FieldsIO &f, const Grid &g, const StepConst &c, int tile_z, cudaStream_t stream,
                             int zb, int ze) {
    using C = V5Cfg<W>;
    cudaError_t e = cudaFuncSetAttribute(step_v5_kernel<FLAGS, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    const int lz = v5_default_lz<W>(g, tile_z, ze - zb);
    const dim3 grid(g.nx / C::WX, g.ny / W, (ze - zb + lz - 1) / lz);
    step_v5_kernel<FLAGS, W><<<grid, C::THREADS, C::SMEM, stream>>>(f, g, c, lz, zb, ze);
    return cudaGetLastError();
}

template <int FLAGS>
cudaError_t launch_step_v5(const FieldsIO &f, const Grid &g, const StepConst &c, int w, int tile_z, cudaStream_t stream,
                           int zb, int ze) {
    if (w == 16) return launch_step_v5_w<FLAGS, 16>(f, g, c, tile_z, stream, zb, ze);
    return launch_step_v5_w<FLAGS, 8>(f, g, c, tile_z, stream, zb, ze);
}

}  // namespace aton
