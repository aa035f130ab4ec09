// The HLL intercell flux (reading S20), tiled and PACKED: step_hll_pk_kernel.
//
// The structure of step_hll_tiled_kernel (aton_step_hll.cuh) -- a CTA owns a tile of columns and marches through a z chunk,
// every cell closed once per plane, records through shared memory, z faces from registers, the product path's chemistry --
// with two x-adjacent cells per thread on the packed fp32x2 forms (aton_pk.cuh): a 64 x 8 tile per 256 threads.
//  * x faces: with own = the thread's pair (cells 2t, 2t+1), Fa = the faces at (2t - 1/2, 2t + 1/2) is one packed face
//    between the pair shifted left by a cell and own, Fb = the faces at (2t + 1/2, 2t + 3/2) one between own and the pair
//    shifted right: U -= mu (Fb - Fa).  The shifted pairs are read from the records cell by cell;
//  * y faces: between own and the same pair of the row below / above (8-byte record reads); z faces from registers;
//  * the tile's ring: the rows below / above as 32 pairs each (warps 0, 1), the cells left / right of each row as one odd
//    pair per row (8 lanes of warp 2).
//  * no plain global load in the loop (the lesson of variant 5, profiles/r02_d_step_v5.md): (N, G) of the next plane -- own
//    pair and ring duty -- are staged by cp.async into thread-private double-buffered slots, x, T, n_H and the source word of
//    the plane being finished into single ones; the records are double buffered by plane parity: one barrier per plane.
// Same formulas as hll_cell / hll_speeds / hll_face (aton_step_ref.cuh); 1/(lambda+ - lambda-) by rcp.approx.
#pragma once
#include "aton_step_fused.cuh"

namespace aton {

__device__ __forceinline__ void cp_async8(void *smem, const void *gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ f2 fmax2(f2 a, f2 b) { return pk(fmaxf(lo(a), lo(b)), fmaxf(hi(a), hi(b))); }
__device__ __forceinline__ f2 fmin2(f2 a, f2 b) { return pk(fminf(lo(a), lo(b)), fminf(hi(a), hi(b))); }

struct HllPair {
    f2 U[4];           // N, Gx, Gy, Gz
    f2 a, s;           // P_dj = a delta_dj + s G_d G_j
};
struct HllSpeeds {     // lambda- and lambda+ along x, y, z in units of c
    f2 lo[3], hi[3];
};

// closure and wave speeds of a pair (hll_cell + hll_speeds<0..2> of aton_step_ref.cuh, packed)
__device__ __forceinline__ void hll_pair(f2 N, f2 gx, f2 gy, f2 gz, HllPair &c, HllSpeeds &w) {
    c.U[0] = N; c.U[1] = gx; c.U[2] = gy; c.U[3] = gz;
    closure2(N, gx, gy, gz, c.a, c.s);
    const float n0 = lo(N), n1 = hi(N);
    const f2 inv = pk(n0 > N_TINY ? m_rcp(n0) : 0.0f, n1 > N_TINY ? m_rcp(n1) : 0.0f);
    f2 r[3] = {gx * inv, gy * inv, gz * inv};
    f2 ff = fma2(r[0], r[0], fma2(r[1], r[1], r[2] * r[2]));
    {   // f > 1 (round-off): rescale the direction ratios, clamp (reading S2)
        const float f0 = lo(ff), f1 = hi(ff);
        const f2 sc = pk(f0 > 1.0f ? rsqrtf(f0) : 1.0f, f1 > 1.0f ? rsqrtf(f1) : 1.0f);
        r[0] = r[0] * sc; r[1] = r[1] * sc; r[2] = r[2] * sc;
        ff = min2(ff, 1.0f);
    }
    const f2 xi = sqrt2(fma2(ff, -3.0f, 4.0f));
    // disc = g [ 2 xi/(xi + 1) - 2 r_d^2/(2 - f^2 + xi) ],  g = 1 - f^2
    const f2 g = 1.0f - ff;
    const f2 A = (xi * 2.0f) * rcp2(xi + 1.0f);
    const f2 B = rcp2((2.0f - ff) + xi) * 2.0f;
    const f2 ixi = rcp2(xi);
#pragma unroll
    for (int d = 0; d < 3; d++) {
        const f2 disc = g * (A - (r[d] * r[d]) * B);
        const f2 root = sqrt2(max2(disc, 0.0f));
        w.lo[d] = (r[d] - root) * ixi;
        w.hi[d] = (r[d] + root) * ixi;
    }
}

// the HLL face flux between pair l (at -e_D) and pair r (at +e_D), half by half (hll_face of aton_step_ref.cuh)
template <int D>
__device__ __forceinline__ void hll_face2(const HllPair &l, f2 lol, f2 hil, const HllPair &r, f2 lor, f2 hir, f2 out[4]) {
    f2 Fl[4], Fr[4];
    flux_row(D, l.U, l.a, l.s, Fl);
    flux_row(D, r.U, r.a, r.s, Fr);
    const f2 sp = max2(fmax2(hil, hir), 0.0f), sm = min2(fmin2(lol, lor), 0.0f);
    const f2 den = sp - sm;
    const float d0 = lo(den), d1 = hi(den);
    const f2 inv = pk(d0 > 0.0f ? m_rcp(d0) : 0.0f, d1 > 0.0f ? m_rcp(d1) : 0.0f);
    const f2 spm = sp * sm;
#pragma unroll
    for (int v = 0; v < 4; v++) out[v] = ((sp * Fl[v] - sm * Fr[v]) + spm * (r.U[v] - l.U[v])) * inv;
    if (!(d0 > 0.0f) || !(d1 > 0.0f)) {        // lambda+ = lambda- = 0 (two beams across the face): the plain average
#pragma unroll
        for (int v = 0; v < 4; v++) {
            const f2 avg = (Fl[v] + Fr[v]) * 0.5f;
            out[v] = pk(d0 > 0.0f ? lo(out[v]) : lo(avg), d1 > 0.0f ? hi(out[v]) : hi(avg));
        }
    }
}

#ifndef HLLPK_DB
#define HLLPK_DB 1       // 1: records double buffered by plane parity (one barrier per plane, 83 KB: 2 CTAs per SM); 0: two barriers
#endif
#ifndef HLLPK_MINB
#define HLLPK_MINB 2     // 116 registers, no spills, 16 warps per SM: 3.2 ms per 512^3 step (3 CTAs at 80 registers with single-buffered records: 4.4 ms)
#endif
struct HllPk {
    static constexpr int TXP = 32, TX = 2 * TXP, TY = 8, SY = TY + 2;
    static constexpr int RS = TX + 4;            // record row: col 1 = the cell left of the tile, cols 2 .. TX + 1 the tile, col TX + 2 the cell right of it
    static constexpr int NREC = 10;              // U0..U3, a, s, lo_x, hi_x, lo_y, hi_y
    static constexpr int PLANE = SY * RS;
    static constexpr int THREADS = TXP * TY;
    static constexpr int NRING = 2 * TXP + TY;   // threads with a ring duty: the two ring rows (a pair each), one odd pair per tile row
    static constexpr int NBUF = HLLPK_DB ? 2 : 1; // record buffers
    static constexpr size_t SMEM = (size_t)NBUF * NREC * PLANE * sizeof(float)
                                   + (size_t)(2 * 4 * THREADS + 2 * 4 * NRING + 4 * THREADS) * sizeof(float2);
};

template <int FLAGS>
__global__ void __launch_bounds__(HllPk::THREADS, HLLPK_MINB) step_hll_pk_kernel(FieldsIO f, Grid g, StepConst c, int lz, int zb, int ze) {
    using C = HllPk;
    extern __shared__ __align__(16) float hsm[];
    float (*rec)[C::NREC][C::PLANE] = reinterpret_cast<float (*)[C::NREC][C::PLANE]>(hsm);          // [NBUF]
    float2 *stg = reinterpret_cast<float2 *>(hsm + C::NBUF * C::NREC * C::PLANE);                     // [2][4][THREADS]: own N, G of the next plane
    float2 *rstg = stg + 2 * 4 * C::THREADS;                                                          // [2][4][NRING]: ring duty
    float2 *xts = rstg + 2 * 4 * C::NRING;                                                            // [4][THREADS]: x, T, n_H, source word
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int x0 = blockIdx.x * C::TX, y0 = blockIdx.y * C::TY, z0 = zb + blockIdx.z * lz;
    const int lzn = min(lz, ze - z0);      // planes [zb, ze): the periodic grid, or a slab's own planes between its ghost planes
    const int plane = g.nx * g.ny;
    const int own = (ty + 1) * C::RS + 2 + 2 * tx;                  // the pair's lo cell in the record frame (even: 8-byte aligned)
    const int col = (y0 + ty) * g.nx + x0 + 2 * tx;                 // ... inside a plane
    // ring duty: warps 0 / 1 the rows below / above the tile (a pair per lane), lanes 0 .. 7 of warp 2 the two cells left and
    // right of tile row `tx`
    const int jb = y0 == 0 ? g.ny - 1 : y0 - 1, jt = y0 + C::TY == g.ny ? 0 : y0 + C::TY;
    const int il = x0 == 0 ? g.nx - 1 : x0 - 1, ir = x0 + C::TX == g.nx ? 0 : x0 + C::TX;
    const bool ring_row = ty < 2, ring_col = ty == 2 && tx < C::TY;
    const int rrow_col = (ty == 0 ? jb : jt) * g.nx + x0 + 2 * tx;
    const int rrow_slot = (ty == 0 ? 0 : C::SY - 1) * C::RS + 2 + 2 * tx;
    const int rcol_l = (y0 + tx) * g.nx + il, rcol_r = (y0 + tx) * g.nx + ir;   // (tx < TY only)
    const int rcol_slot = (tx + 1) * C::RS;                          // + 1: left cell, + TX + 2: right cell

    const int rix = ty < 2 ? threadIdx.x : 2 * C::TXP + tx;          // ring duty index (ring_row / ring_col threads)
    int par = 0;                                                    // record buffer of the plane being formed
    auto put2 = [&](int r, int slot, f2 v) { *reinterpret_cast<float2 *>(&rec[par][r][slot]) = make_float2(lo(v), hi(v)); };
    auto get2 = [&](int r, int slot) { const float2 v = *reinterpret_cast<const float2 *>(&rec[par][r][slot]); return pk(v.x, v.y); };
    auto get11 = [&](int r, int slot) { return pk(rec[par][r][slot], rec[par][r][slot + 1]); };      // a pair at an odd column
    auto sget = [&](const float2 *p) { const float2 v = *p; return pk(v.x, v.y); };
    const float *src[4] = {f.N, f.Gx, f.Gy, f.Gz};
    // stage plane kk into buffer b: the thread's own pair, and its ring duty if the plane belongs to the chunk
    auto stage = [&](int b, int kk, bool inp) {
        float2 *d = stg + (size_t)b * 4 * C::THREADS + threadIdx.x;
        const int base = kk * plane;
#pragma unroll
        for (int v = 0; v < 4; v++) cp_async8(d + v * C::THREADS, src[v] + base + col);
        if (inp) {
            float2 *rd = rstg + (size_t)b * 4 * C::NRING + rix;
            if (ring_row) {
#pragma unroll
                for (int v = 0; v < 4; v++) cp_async8(rd + v * C::NRING, src[v] + base + rrow_col);
            } else if (ring_col) {
#pragma unroll
                for (int v = 0; v < 4; v++) {
                    cp_async4(reinterpret_cast<float *>(rd + v * C::NRING), src[v] + base + rcol_l);
                    cp_async4(reinterpret_cast<float *>(rd + v * C::NRING) + 1, src[v] + base + rcol_r);
                }
            }
        }
        cp_async_commit();
    };

    const float mu = 2.0f * c.h;                                    // c dt / dx
    const f2 zero = splat(0.0f);
    HllPair prev;                                                   // the column pair's cells in plane m-1, their z speeds
    f2 ploz = zero, phiz = zero;
    f2 Unp[4] = {zero, zero, zero, zero};                           // plane m-1 after its x and y faces
    f2 Fzb[4] = {zero, zero, zero, zero};                           // the face below plane m-1
#pragma unroll
    for (int v = 0; v < 4; v++) prev.U[v] = zero;
    prev.a = zero; prev.s = zero;
    int idp = 0;
    int k = z0 == 0 ? g.nz - 1 : z0 - 1;
    stage(0, k, false);
    for (int m = 0; m <= lzn + 1; m++) {
        const bool inpl = m >= 1 && m <= lzn;                       // plane m belongs to the chunk (CTA-uniform)
        const int id = k * plane + col;
        const int kn = k + 1 == g.nz ? 0 : k + 1;
        const int sb_ = m & 1;                                      // staging buffer of plane m
        par = HLLPK_DB ? sb_ : 0;
        cp_async_wait_all();                                        // this thread's part of plane m has landed
        const float2 *sd = stg + (size_t)sb_ * 4 * C::THREADS + threadIdx.x;
        HllPair ce;
        HllSpeeds w;
        hll_pair(sget(sd), sget(sd + C::THREADS), sget(sd + 2 * C::THREADS), sget(sd + 3 * C::THREADS), ce, w);
        HllPair rc;                                                 // ring duty of plane m (read before the slots are re-staged)
        HllSpeeds rw;
        if (inpl && (ring_row || ring_col)) {
            const float2 *rd = rstg + (size_t)sb_ * 4 * C::NRING + rix;
            hll_pair(sget(rd), sget(rd + C::NRING), sget(rd + 2 * C::NRING), sget(rd + 3 * C::NRING), rc, rw);
        }
        // x, T, n_H and the source word of plane m-1 (finished at the end of this iteration), then the next plane's staging
        const bool fin = m >= 2;
        if (fin) {
            float2 *xd = xts + threadIdx.x;
            cp_async8(xd, f.x + idp);
            cp_async8(xd + C::THREADS, f.T + idp);
            cp_async8(xd + 2 * C::THREADS, f.nH + idp);
            cp_async4(reinterpret_cast<float *>(xd + 3 * C::THREADS), f.src_bits + ((unsigned)idp >> 5));
            cp_async_commit();
        }
        const bool more = m <= lzn;
        if (more) stage(sb_ ^ 1, kn, m + 1 <= lzn);
        f2 Un[4] = {ce.U[0], ce.U[1], ce.U[2], ce.U[3]};
        if (inpl) {
            // ---- publish the records of the tile and of its ring
#pragma unroll
            for (int v = 0; v < 4; v++) put2(v, own, ce.U[v]);
            put2(4, own, ce.a); put2(5, own, ce.s);
            put2(6, own, w.lo[0]); put2(7, own, w.hi[0]); put2(8, own, w.lo[1]); put2(9, own, w.hi[1]);
            if (ring_row) {
#pragma unroll
                for (int v = 0; v < 4; v++) put2(v, rrow_slot, rc.U[v]);
                put2(4, rrow_slot, rc.a); put2(5, rrow_slot, rc.s);
                put2(8, rrow_slot, rw.lo[1]); put2(9, rrow_slot, rw.hi[1]);
            } else if (ring_col) {
                const int sl = rcol_slot + 1, sr = rcol_slot + C::TX + 2;
#pragma unroll
                for (int v = 0; v < 4; v++) { rec[par][v][sl] = lo(rc.U[v]); rec[par][v][sr] = hi(rc.U[v]); }
                rec[par][4][sl] = lo(rc.a); rec[par][4][sr] = hi(rc.a);
                rec[par][5][sl] = lo(rc.s); rec[par][5][sr] = hi(rc.s);
                rec[par][6][sl] = lo(rw.lo[0]); rec[par][6][sr] = hi(rw.lo[0]);
                rec[par][7][sl] = lo(rw.hi[0]); rec[par][7][sr] = hi(rw.hi[0]);
            }
            __syncthreads();      // (with double-buffered records the one barrier of the plane: buffer `par` is not written again
                                  // before every warp has passed the barrier of plane m+1)
            // ---- x: Fa between the pair shifted left by a cell and own, Fb between own and the pair shifted right
            {
                HllPair nb;
                f2 Fa[4], Fb[4];
#pragma unroll
                for (int v = 0; v < 4; v++) nb.U[v] = get11(v, own - 1);
                nb.a = get11(4, own - 1); nb.s = get11(5, own - 1);
                hll_face2<0>(nb, get11(6, own - 1), get11(7, own - 1), ce, w.lo[0], w.hi[0], Fa);
#pragma unroll
                for (int v = 0; v < 4; v++) nb.U[v] = get11(v, own + 1);
                nb.a = get11(4, own + 1); nb.s = get11(5, own + 1);
                hll_face2<0>(ce, w.lo[0], w.hi[0], nb, get11(6, own + 1), get11(7, own + 1), Fb);
#pragma unroll
                for (int v = 0; v < 4; v++) Un[v] = Un[v] - (Fb[v] - Fa[v]) * mu;
            }
            // ---- y: the same pair of the row below and of the row above
            {
                HllPair nb;
                f2 Fa[4], Fb[4];
#pragma unroll
                for (int v = 0; v < 4; v++) nb.U[v] = get2(v, own - C::RS);
                nb.a = get2(4, own - C::RS); nb.s = get2(5, own - C::RS);
                hll_face2<1>(nb, get2(8, own - C::RS), get2(9, own - C::RS), ce, w.lo[1], w.hi[1], Fa);
#pragma unroll
                for (int v = 0; v < 4; v++) nb.U[v] = get2(v, own + C::RS);
                nb.a = get2(4, own + C::RS); nb.s = get2(5, own + C::RS);
                hll_face2<1>(ce, w.lo[1], w.hi[1], nb, get2(8, own + C::RS), get2(9, own + C::RS), Fb);
#pragma unroll
                for (int v = 0; v < 4; v++) Un[v] = Un[v] - (Fb[v] - Fa[v]) * mu;
            }
        }
        if (m >= 1) {
            f2 Fz[4];                                               // the face between planes m-1 and m
            hll_face2<2>(prev, ploz, phiz, ce, w.lo[2], w.hi[2], Fz);
            if (fin) {                                              // plane m-1 is complete: chemistry, store
#pragma unroll
                for (int v = 0; v < 4; v++) Unp[v] = Unp[v] - (Fz[v] - Fzb[v]) * mu;
                // one straight-line chemistry sub-step; a source cell, or a cell that needs sub-cycling, keeps its transported
                // values and is flagged for step_fixup_kernel / step_stiff_kernel, as in variants 4 and 5
                if (more) cp_async_wait_1(); else cp_async_wait_all();     // the next plane's staging may still fly
                const float2 *xd = xts + threadIdx.x;
                f2 x2 = sget(xd), T2 = sget(xd + C::THREADS);
                const f2 h2 = sget(xd + 2 * C::THREADS);
                const unsigned sw = *reinterpret_cast<const unsigned *>(xd + 3 * C::THREADS);
                const unsigned sb = (sw >> (idp & 31)) & 3u;
                const unsigned d = chem_fast2<FLAGS>(Unp[0], Unp[1], Unp[2], Unp[3], x2, T2, h2, c, sb);
#define ATON_ST2(ptr, A) *reinterpret_cast<float2 *>(ptr + idp) = make_float2(lo(A), hi(A))
                ATON_ST2(f.N1, Unp[0]); ATON_ST2(f.Gx1, Unp[1]); ATON_ST2(f.Gy1, Unp[2]); ATON_ST2(f.Gz1, Unp[3]);
                ATON_ST2(f.x, x2); ATON_ST2(f.T, T2);
#undef ATON_ST2
                if (d) atomicOr(f.defer_mask + ((unsigned)idp >> 5), d << (idp & 31));
            }
#pragma unroll
            for (int v = 0; v < 4; v++) Fzb[v] = Fz[v];
        }
        prev = ce; ploz = w.lo[2]; phiz = w.hi[2];
#pragma unroll
        for (int v = 0; v < 4; v++) Unp[v] = Un[v];
        idp = id;
        k = kn;
#if !HLLPK_DB
        if (inpl) __syncthreads();                                  // the records are overwritten by the next plane
#endif
    }
}

inline bool hll_pk_grid_ok(const Grid &g) { return g.nx % HllPk::TX == 0 && g.ny % HllPk::TY == 0; }

template <int FLAGS>
cudaError_t launch_step_hll_pk(const FieldsIO &f, const Grid &g, const StepConst &c, cudaStream_t stream, int zb, int ze) {
    const int nzr = ze - zb;
    const long tiles_xy = (long)(g.nx / HllPk::TX) * (g.ny / HllPk::TY);
    int lz = 32;      // largest power of two <= 32 that still gives >= 4 waves of 4 CTAs per SM
    while (lz > 4 && tiles_xy * ((nzr + lz - 1) / lz) < 4L * 4 * 148) lz >>= 1;
    lz = lz < nzr ? lz : nzr;
    const dim3 grid(g.nx / HllPk::TX, g.ny / HllPk::TY, (nzr + lz - 1) / lz);
    cudaError_t e = cudaFuncSetAttribute(step_hll_pk_kernel<FLAGS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)HllPk::SMEM);
    if (e != cudaSuccess) return e;
    step_hll_pk_kernel<FLAGS><<<grid, HllPk::THREADS, HllPk::SMEM, stream>>>(f, g, c, lz, zb, ze);
    return cudaGetLastError();
}

}  // namespace aton
