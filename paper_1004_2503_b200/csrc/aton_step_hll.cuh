// The HLL intercell flux (reading S20) as a tiled kernel: step_hll_tiled_kernel.
//
// step_hll_kernel (aton_step_ref.cuh) is the by-eye statement: one thread per cell closes its six neighbours again and
// evaluates the wave speeds of both cells of each of its six faces -- seven closures, twelve speed pairs, 28 global loads
// per cell.  Here a CTA owns a 32 x 8 tile of columns and marches through a z chunk:
//  * every cell of the tile and of its one-cell ring is closed ONCE per plane, its wave speeds along x and y evaluated once,
//    and the record (U, a, s, lambda-_x, lambda+_x, lambda-_y, lambda+_y) published to shared memory (340 records, 13.6 KB);
//  * a thread forms the four lateral faces of its cell from the records (each lateral face is formed by both of its cells:
//    no second barrier), the z faces from registers -- the column's previous cell and its z speeds are carried, and the
//    face between planes m-1 and m closes plane m-1 and opens plane m;
//  * the same device functions in the same order as step_hll_kernel (x, then y, then z; hll_cell, hll_speeds, the face
//    formula): the two kernels agree to rounding (the compiler contracts the face formula differently in the two);
//  * the chemistry is the product path's: one straight-line sub-step (chem_fast2), source cells and cells that need
//    sub-cycling flagged in the mask for step_fixup_kernel / step_stiff_kernel (fp64).
// Grids it tiles: nx % 32 == 0 and ny % 8 == 0 with kernel variant 4 or 5 selected; everything else runs step_hll_kernel.
#pragma once
#include "aton_physics_pk.cuh"
#include "aton_step_ref.cuh"

namespace aton {

// the face formula of hll_face with the wave speeds of both cells given (hll_face evaluates them itself)
template <int D>
__device__ __forceinline__ void hll_face_pre(const HllCell &l, float lol, float hil, const HllCell &r, float lor, float hir,
                                             float out[4]) {
    float Fl[4], Fr[4];
    hll_flux_row<D>(l, Fl);
    hll_flux_row<D>(r, Fr);
    const float sp = fmaxf(0.0f, fmaxf(hil, hir)), sm = fminf(0.0f, fminf(lol, lor));
    const float den = sp - sm;
    if (den > 0.0f) {
        const float inv = 1.0f / den, spm = sp * sm;
#pragma unroll
        for (int v = 0; v < 4; v++) out[v] = (sp * Fl[v] - sm * Fr[v] + spm * (r.U[v] - l.U[v])) * inv;
    } else {
#pragma unroll
        for (int v = 0; v < 4; v++) out[v] = 0.5f * (Fl[v] + Fr[v]);
    }
}

struct HllTile {
    static constexpr int TX = 32, TY = 8, SX = TX + 2, SY = TY + 2, NC = SX * SY, NREC = 10, THREADS = TX * TY;
};

template <int FLAGS>
__global__ void __launch_bounds__(HllTile::THREADS) step_hll_tiled_kernel(FieldsIO f, Grid g, StepConst c, int lz, int zb, int ze) {
    using C = HllTile;
    __shared__ float rec[C::NREC][C::NC];     // U0..U3, a, s, lo_x, hi_x, lo_y, hi_y of the tile and its ring, current plane
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int x0 = blockIdx.x * C::TX, y0 = blockIdx.y * C::TY, z0 = zb + blockIdx.z * lz;
    const int lzn = min(lz, ze - z0);      // planes [zb, ze): the periodic grid, or a slab's own planes between its ghost planes
    const int plane = g.nx * g.ny;
    const int own = (ty + 1) * C::SX + tx + 1;                      // this thread's cell in the record frame
    const int col = (y0 + ty) * g.nx + x0 + tx;                     // ... inside a plane
    // ring cell of threads 0 .. 83: rows sy = 0 and SY - 1 (34 each), columns sx = 0 and SX - 1 (8 each)
    const int h = threadIdx.x;
    const bool ring = h < 2 * C::SX + 2 * C::TY;
    int rsx = 0, rsy = 0;
    if (h < C::SX) { rsx = h; rsy = 0; }
    else if (h < 2 * C::SX) { rsx = h - C::SX; rsy = C::SY - 1; }
    else if (h < 2 * C::SX + C::TY) { rsx = 0; rsy = 1 + h - 2 * C::SX; }
    else { rsx = C::SX - 1; rsy = 1 + h - 2 * C::SX - C::TY; }
    int gi = x0 - 1 + rsx, gj = y0 - 1 + rsy;
    gi += gi < 0 ? g.nx : 0; gi -= gi >= g.nx ? g.nx : 0;
    gj += gj < 0 ? g.ny : 0; gj -= gj >= g.ny ? g.ny : 0;
    const int rcol = gj * g.nx + gi, rslot = rsy * C::SX + rsx;

    auto publish = [&](int slot, const HllCell &ce) {
        float lox, hix, loy, hiy;
        hll_speeds<0>(ce, lox, hix);
        hll_speeds<1>(ce, loy, hiy);
        rec[0][slot] = ce.U[0]; rec[1][slot] = ce.U[1]; rec[2][slot] = ce.U[2]; rec[3][slot] = ce.U[3];
        rec[4][slot] = ce.a; rec[5][slot] = ce.s;
        rec[6][slot] = lox; rec[7][slot] = hix; rec[8][slot] = loy; rec[9][slot] = hiy;
    };
    // a neighbour as the face formula needs it (U, a, s; the speeds come separately)
    auto fetch = [&](int slot, HllCell &nb) {
        nb.U[0] = rec[0][slot]; nb.U[1] = rec[1][slot]; nb.U[2] = rec[2][slot]; nb.U[3] = rec[3][slot];
        nb.a = rec[4][slot]; nb.s = rec[5][slot];
    };

    const float mu = 2.0f * c.h;                                   // c dt / dx
    HllCell prev;                                                  // the column's cell in plane m-1, its z speeds
    float ploz = 0.f, phiz = 0.f;
    float Unp[4] = {0.f, 0.f, 0.f, 0.f};                           // plane m-1 after its x and y faces
    float Fzb[4] = {0.f, 0.f, 0.f, 0.f};                           // the face below plane m-1
    int idp = 0;
    int k = z0 == 0 ? g.nz - 1 : z0 - 1;
    for (int m = 0; m <= lzn + 1; m++) {
        const bool inpl = m >= 1 && m <= lzn;                      // plane m belongs to the chunk (CTA-uniform)
        const int id = k * plane + col;
        HllCell ce;
        hll_cell(__ldg(f.N + id), __ldg(f.Gx + id), __ldg(f.Gy + id), __ldg(f.Gz + id), ce);
        float loz, hiz;
        hll_speeds<2>(ce, loz, hiz);
        float Un[4] = {ce.U[0], ce.U[1], ce.U[2], ce.U[3]};
        if (inpl) {
            publish(own, ce);
            if (ring) {
                const int rid = k * plane + rcol;
                HllCell rc;
                hll_cell(__ldg(f.N + rid), __ldg(f.Gx + rid), __ldg(f.Gy + rid), __ldg(f.Gz + rid), rc);
                publish(rslot, rc);
            }
            __syncthreads();
            const float lox = rec[6][own], hix = rec[7][own], loy = rec[8][own], hiy = rec[9][own];
            HllCell nb;
            float fhi[4], flo[4];
            fetch(own + 1, nb);
            hll_face_pre<0>(ce, lox, hix, nb, rec[6][own + 1], rec[7][own + 1], fhi);
            fetch(own - 1, nb);
            hll_face_pre<0>(nb, rec[6][own - 1], rec[7][own - 1], ce, lox, hix, flo);
#pragma unroll
            for (int v = 0; v < 4; v++) Un[v] -= mu * (fhi[v] - flo[v]);
            fetch(own + C::SX, nb);
            hll_face_pre<1>(ce, loy, hiy, nb, rec[8][own + C::SX], rec[9][own + C::SX], fhi);
            fetch(own - C::SX, nb);
            hll_face_pre<1>(nb, rec[8][own - C::SX], rec[9][own - C::SX], ce, loy, hiy, flo);
#pragma unroll
            for (int v = 0; v < 4; v++) Un[v] -= mu * (fhi[v] - flo[v]);
        }
        if (m >= 1) {
            float Fz[4];                                           // the face between planes m-1 and m
            hll_face_pre<2>(prev, ploz, phiz, ce, loz, hiz, Fz);
            if (m >= 2) {                                          // plane m-1 is complete: chemistry, store
#pragma unroll
                for (int v = 0; v < 4; v++) Unp[v] -= mu * (Fz[v] - Fzb[v]);
                // one straight-line chemistry sub-step (chem_fast2 on a splat pair: the packed form costs the issue slots
                // of the scalar one); a source cell, or a cell that needs sub-cycling, keeps its transported values and is
                // flagged for step_fixup_kernel / step_stiff_kernel, as in variants 4 and 5
                const unsigned sb = (__ldg(f.src_bits + ((unsigned)idp >> 5)) >> (idp & 31)) & 1u;
                f2 N2 = splat(Unp[0]), gx2 = splat(Unp[1]), gy2 = splat(Unp[2]), gz2 = splat(Unp[3]);
                f2 x2 = splat(f.x[idp]), T2 = splat(f.T[idp]);
                const unsigned d = chem_fast2<FLAGS>(N2, gx2, gy2, gz2, x2, T2, splat(__ldg(f.nH + idp)), c, sb ? 3u : 0u);
                f.N1[idp] = lo(N2); f.Gx1[idp] = lo(gx2); f.Gy1[idp] = lo(gy2); f.Gz1[idp] = lo(gz2);
                f.x[idp] = lo(x2); f.T[idp] = lo(T2);
                if (d & 1u) atomicOr(f.defer_mask + ((unsigned)idp >> 5), 1u << (idp & 31));
            }
#pragma unroll
            for (int v = 0; v < 4; v++) Fzb[v] = Fz[v];
        }
        prev = ce; ploz = loz; phiz = hiz;
#pragma unroll
        for (int v = 0; v < 4; v++) Unp[v] = Un[v];
        idp = id;
        k = k + 1 == g.nz ? 0 : k + 1;
        if (inpl) __syncthreads();                                 // the records are overwritten by the next plane
    }
}

inline bool hll_tiled_grid_ok(const Grid &g) { return g.nx % HllTile::TX == 0 && g.ny % HllTile::TY == 0; }

template <int FLAGS>
cudaError_t launch_step_hll_tiled(const FieldsIO &f, const Grid &g, const StepConst &c, cudaStream_t stream, int zb, int ze) {
    const int nzr = ze - zb;
    const long tiles_xy = (long)(g.nx / HllTile::TX) * (g.ny / HllTile::TY);
    int lz = 32;      // largest power of two <= 32 that still gives >= 4 waves of 8 CTAs per SM
    while (lz > 4 && tiles_xy * ((nzr + lz - 1) / lz) < 4L * 8 * 148) lz >>= 1;
    lz = lz < nzr ? lz : nzr;
    const dim3 grid(g.nx / HllTile::TX, g.ny / HllTile::TY, (nzr + lz - 1) / lz);
    step_hll_tiled_kernel<FLAGS><<<grid, HllTile::THREADS, 0, stream>>>(f, g, c, lz, zb, ze);
    return cudaGetLastError();
}

}  // namespace aton
