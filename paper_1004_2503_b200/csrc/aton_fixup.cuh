// The cells the fused step kernels do not finish: cells that need more than one chemistry sub-cycle (the Anninos
// 10 % rule, reading S5; "sub-cycled", L442 "branching has some impact on the performance")
// and, for variant 4, the source cells.  They hold their transported (N, G) and their old (x, T).
//
//  * variant 4 (product): the warp that produced a cell redoes it itself.  The ids of deferred cells go into a
//    warp-private shared-memory queue; whenever it holds 32 the whole warp runs the sub-cycled fp32 operator on 32
//    cells at once (v4_fix_drain), reading and writing lines the same warp wrote moments ago -- they are still in
//    L2, so the redo costs no extra HBM traffic and no mask scan.  A cell whose fp32 sub-cycling reports
//    cancellation (chemistry<.., BAIL>) is appended to a small global queue and redone in fp64 by step_stiff_kernel.
//  * variant 2 (fallback grids): step_fixup_kernel scans a 1-bit-per-cell mask and redoes the flagged cells
//    (fp32, fp64 redo inline).
// stats[0] += sum(nsub - 1), stats[1] = max nsub, stats[2] += cells redone, stats[3] += cells redone in fp64.
#pragma once
#include "aton_step_ref.cuh"

namespace aton {

// what the cold paths need, in global memory (kernel parameters cannot be passed on by address without a local copy)
struct FixArgs {
    FieldsIO f;
    StepConst c;
    StepConstD cd;
};

constexpr int V4_QCAP = 160;                // ids per warp queue: < 32 left over + up to 128 new per plane
constexpr int V4_QWORDS = V4_QCAP + 32;     // + 4 statistics words (+ padding to keep 128-byte alignment)

// Redo queued cells, 32 at a time from the END of the queue, while it holds at least `thresh` ids; returns what is left.
// A cell's transported (N, G) and old (x, T) are read back from global memory (the owner lane wrote them moments ago:
// L2 hits; the caller's __syncwarp orders those stores before these loads).
template <int FLAGS>
__device__ __noinline__ int v4_fix_drain(const FixArgs *fa, int *q, int qn, int thresh) {
    const int lane = threadIdx.x & 31;
    int *wst = q + V4_QCAP;
    const FieldsIO &f = fa->f;
    while (qn >= thresh && qn > 0) {
        const int n = min(qn, 32);
        qn -= n;
        if (lane < n) {
            const int id = q[qn + lane];
            float N = f.N1[id], gx = f.Gx1[id], gy = f.Gy1[id], gz = f.Gz1[id], x = f.x[id], T = f.T[id];
            const float nH = __ldg(f.nH + id);
            if ((__ldg(f.src_bits + ((unsigned)id >> 5)) >> (id & 31)) & 1u) N += source_lookup(f, id, fa->c.dt);
            const int ns = chemistry<FLAGS, true>(N, gx, gy, gz, x, T, nH, fa->c);
            if (ns >= 0) {
                f.N1[id] = N; f.Gx1[id] = gx; f.Gy1[id] = gy; f.Gz1[id] = gz;
                f.x[id] = x; f.T[id] = T;
                atomicAdd(wst, ns - 1);
                atomicMax(wst + 1, ns);
                atomicAdd(wst + 2, 1);
            } else {        // stiff: the cell keeps its values; the fp64 kernel redoes it from them
                const unsigned slot = atomicAdd(f.stiff_n, 1u);
                if (slot < f.stiff_cap) {
                    f.stiff_q[slot] = id;
                } else {    // queue full (the cap is ncell / 16): redo it here
                    double Nd = (double)f.N1[id] + source_lookup_d(f, id, fa->cd.dt), ax = f.Gx1[id], ay = f.Gy1[id], az = f.Gz1[id];
                    double xd = f.x[id], Td = f.T[id];
                    const int nd = chemistry_f64<FLAGS>(Nd, ax, ay, az, xd, Td, (double)nH, fa->cd);
                    f.N1[id] = (float)Nd; f.Gx1[id] = (float)ax; f.Gy1[id] = (float)ay; f.Gz1[id] = (float)az;
                    f.x[id] = (float)xd; f.T[id] = (float)Td;
                    atomicAdd(wst, nd - 1);
                    atomicMax(wst + 1, nd);
                    atomicAdd(wst + 2, 1);
                    atomicAdd(wst + 3, 1);
                }
            }
        }
        __syncwarp();
    }
    return qn;
}

// fp64 redo of the cells queued by v4_fix_drain; also re-arms the queue counter for the next step
template <int FLAGS>
__global__ void __launch_bounds__(128) step_stiff_kernel(const FixArgs *fa) {
    const FieldsIO &f = fa->f;
    const unsigned n = min(f.stiff_n[0], f.stiff_cap);
    int extra = 0, mx = 0, cells = 0;
    for (unsigned e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
        const int id = f.stiff_q[e];
        double N = f.N1[id], gx = f.Gx1[id], gy = f.Gy1[id], gz = f.Gz1[id], x = f.x[id], T = f.T[id];
        if ((__ldg(f.src_bits + ((unsigned)id >> 5)) >> (id & 31)) & 1u) N += source_lookup_d(f, id, fa->cd.dt);
        const int ns = chemistry_f64<FLAGS>(N, gx, gy, gz, x, T, (double)__ldg(f.nH + id), fa->cd);
        f.N1[id] = (float)N; f.Gx1[id] = (float)gx; f.Gy1[id] = (float)gy; f.Gz1[id] = (float)gz;
        f.x[id] = (float)x; f.T[id] = (float)T;
        extra += ns - 1; mx = max(mx, ns); cells++;
    }
    for (int o = 16; o > 0; o >>= 1) {
        extra += __shfl_xor_sync(0xffffffffu, extra, o);
        cells += __shfl_xor_sync(0xffffffffu, cells, o);
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((threadIdx.x & 31) == 0 && cells > 0) {
        atomicAdd(f.stats, (unsigned long long)extra);
        atomicMax(f.stats + 1, (unsigned long long)mx);
        atomicAdd(f.stats + 2, (unsigned long long)cells);
        atomicAdd(f.stats + 3, (unsigned long long)cells);
    }
    // the last block to finish zeroes the counter ([1] counts finished blocks)
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(f.stiff_n + 1, 1u) == gridDim.x - 1) { f.stiff_n[0] = 0u; f.stiff_n[1] = 0u; }
    }
}

// ---------------------------------------------------------------------------------------------------
// Variant 2's fix-up: the mask is scanned in chunks of 256 words; flagged cells are compacted into a
// shared-memory queue and processed one per thread once the queue holds a few hundred (or the scan ends),
// so the data-dependent sub-cycle loops run on full warps.  Sources were injected by the step kernel.
// ---------------------------------------------------------------------------------------------------
constexpr int FIXUP_THREADS = 256, FIXUP_QTHRESH = 512, FIXUP_QCAP = FIXUP_QTHRESH + 32 * FIXUP_THREADS;

template <int FLAGS>
__global__ void __launch_bounds__(FIXUP_THREADS) step_fixup_kernel(FieldsIO f, StepConst c, StepConstD cd, int nwords) {
    __shared__ int queue[FIXUP_QCAP];
    __shared__ int qn;
    if (threadIdx.x == 0) qn = 0;
    __syncthreads();
    int nsub_extra = 0, nsub_max = 0, ncell = 0, nstiff = 0;
    const int nchunks = (nwords + FIXUP_THREADS - 1) / FIXUP_THREADS;
    for (int ch = blockIdx.x; ch < nchunks + (int)gridDim.x; ch += gridDim.x) {
        const bool scan = ch < nchunks;         // the last trip only drains the queue
        if (scan) {
            const int w = ch * FIXUP_THREADS + threadIdx.x;
            unsigned bits = w < nwords ? f.defer_mask[w] : 0u;
            if (bits) {
                f.defer_mask[w] = 0u;
                int pos = atomicAdd(&qn, __popc(bits));
                while (bits) {
                    const int b = __ffs(bits) - 1;
                    bits &= bits - 1;
                    queue[pos++] = w * 32 + b;
                }
            }
        }
        __syncthreads();
        const int n = qn;
        if (n >= FIXUP_QTHRESH || (!scan && n > 0)) {
            for (int it = threadIdx.x; it < n; it += FIXUP_THREADS) {
                const int id = queue[it];
                float N = f.N1[id], gx = f.Gx1[id], gy = f.Gy1[id], gz = f.Gz1[id];
                float x = f.x[id], T = f.T[id];
                const float nH = __ldg(f.nH + id);
                const float N0 = N, gx0 = gx, gy0 = gy, gz0 = gz, x0 = x, T0 = T;
                int ns = chemistry<FLAGS, true>(N, gx, gy, gz, x, T, nH, c);
                if (ns < 0) {
                    double Nd = N0, ax = gx0, ay = gy0, az = gz0, xd = x0, Td = T0;
                    ns = chemistry_f64<FLAGS>(Nd, ax, ay, az, xd, Td, (double)nH, cd);
                    N = (float)Nd; gx = (float)ax; gy = (float)ay; gz = (float)az; x = (float)xd; T = (float)Td;
                    nstiff++;
                }
                f.N1[id] = N; f.Gx1[id] = gx; f.Gy1[id] = gy; f.Gz1[id] = gz;
                f.x[id] = x; f.T[id] = T;
                nsub_extra += ns - 1;
                nsub_max = max(nsub_max, ns);
                ncell++;
            }
            __syncthreads();
            if (threadIdx.x == 0) qn = 0;
        }
        __syncthreads();
        if (!scan) break;
    }
    // statistics: warp reduce, one atomic set per warp that saw work
    for (int o = 16; o > 0; o >>= 1) {
        nsub_extra += __shfl_xor_sync(0xffffffffu, nsub_extra, o);
        ncell += __shfl_xor_sync(0xffffffffu, ncell, o);
        nstiff += __shfl_xor_sync(0xffffffffu, nstiff, o);
        nsub_max = max(nsub_max, __shfl_xor_sync(0xffffffffu, nsub_max, o));
    }
    if ((threadIdx.x & 31) == 0 && ncell > 0) {
        atomicAdd(f.stats, (unsigned long long)nsub_extra);
        atomicMax(f.stats + 1, (unsigned long long)nsub_max);
        atomicAdd(f.stats + 2, (unsigned long long)ncell);
        atomicAdd(f.stats + 3, (unsigned long long)nstiff);
    }
}

template <int FLAGS>
cudaError_t launch_step_fixup(const FieldsIO &f, const Grid &g, const StepConst &c, const StepConstD &cd, cudaStream_t stream) {
    const long ncell = (long)g.nx * g.ny * g.nz;
    const int nwords = (int)((ncell + 31) / 32);
    const int nchunks = (nwords + FIXUP_THREADS - 1) / FIXUP_THREADS;
    const int blocks = nchunks < 148 * 8 ? nchunks : 148 * 8;
    step_fixup_kernel<FLAGS><<<blocks, FIXUP_THREADS, 0, stream>>>(f, c, cd, nwords);
    return cudaGetLastError();
}

template <int FLAGS>
cudaError_t launch_step_stiff(const FixArgs *fa, cudaStream_t stream) {
    step_stiff_kernel<FLAGS><<<148, 128, 0, stream>>>(fa);
    return cudaGetLastError();
}

}  // namespace aton
