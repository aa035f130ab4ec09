// The cells the fused step kernels do not finish: cells that need more than one chemistry sub-cycle (the Anninos
// 10 % rule, reading S5; "sub-cycled", L442 "branching has some impact on the performance")
// and, for variant 4, the source cells.  They hold their transported (N, G) and their old (x, T) and are flagged in
// a 1-bit-per-cell mask.
//  * step_fixup_kernel scans the mask, compacts the flagged cells into a shared-memory queue and runs the sub-cycled
//    fp32 operator on full warps.  A cell whose fp32 sub-cycling is not accurate enough -- heating and cooling cancel
//    under an active 10 % rule, or the attenuation of N is too sensitive to the sub-step partition (chemistry<.., BAIL>,
//    DESIGN.md 5.3) -- keeps its values and is appended to a global queue of ids;
//  * step_stiff_kernel redoes the queued cells in fp64 (aton_physics_f64.cuh) and re-arms the queue.
// Redoing the deferred cells inside the step kernel instead (warp-private queue, 32 cells at a time, lines still in
// L2) was built and measured in round 2 and lost in every state: profiles/r02_b_fixup.md.
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

// fp64 redo of the cells queued by step_fixup_kernel; also re-arms the queue counter for the next step
template <int FLAGS>
__global__ void __launch_bounds__(128) step_stiff_kernel(const FixArgs *fa) {
    const FieldsIO &f = fa->f;
    const unsigned n = min(f.stiff_n[0], f.stiff_cap);
    int extra = 0, mx = 0, cells = 0;
    for (unsigned e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
        const int id = f.stiff_q[e];
        double N = f.N1[id], gx = f.Gx1[id], gy = f.Gy1[id], gz = f.Gz1[id], x = f.x[id], T = f.T[id];
        if (f.fix_inject && ((__ldg(f.src_bits + ((unsigned)id >> 5)) >> (id & 31)) & 1u)) N += source_lookup_d(f, id, fa->cd.dt);
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
// FIXUP_GROUP chunks of FIXUP_THREADS words are scanned behind one vote: 8 on large grids (an empty scan of 1024^3 costs
// 0.08 ms instead of 0.25), 2 or 1 on small ones so that the groups still outnumber the resident blocks (256^3 has 256
// groups of 8: a block then redoes ~1300 cells, five batches per warp one after the other)

// INLINE64: small grids (<= 2^21 cells) redo their stiff cells here, in place, instead of queueing them for step_stiff_kernel:
// that kernel's launch and 17 us floor are a quarter of a 128^3 step
template <int FLAGS, int FIXUP_GROUP, bool INLINE64>
__global__ void __launch_bounds__(FIXUP_THREADS, INLINE64 ? 2 : 3) step_fixup_kernel(const FixArgs *fa, int word0, int nwords) {
    __shared__ int queue[FIXUP_QCAP];
    __shared__ int qn, qhead;
    const FieldsIO &f = fa->f;
    if (threadIdx.x == 0) { qn = 0; qhead = 0; }
    __syncthreads();
    int nsub_extra = 0, nsub_max = 0, ncell = 0, n64 = 0;
    // redo the queued cells (all threads of the block call this together)
    auto drain = [&]() {
        const int n = qn;
        // self-scheduling by warps: a warp takes the next 32 cells when it is done with its own, so a round lasts as
        // long as its slowest warp, not as long as the slowest cell of every stride (source cells take tens of
        // sub-cycles); one shared-memory atomic per 32 cells
        for (;;) {
            int it = 0;
            if ((threadIdx.x & 31) == 0) it = atomicAdd(&qhead, 32);
            it = __shfl_sync(0xffffffffu, it, 0) + (threadIdx.x & 31);
            if (it - (int)(threadIdx.x & 31) >= n) break;
            if (it >= n) continue;
            const int id = queue[it];
            float N = f.N1[id], gx = f.Gx1[id], gy = f.Gy1[id], gz = f.Gz1[id];
            float x = f.x[id], T = f.T[id];
            if (f.fix_inject && ((__ldg(f.src_bits + ((unsigned)id >> 5)) >> (id & 31)) & 1u)) N += source_lookup(f, id, fa->c.dt);
            const int ns = chemistry<FLAGS, true>(N, gx, gy, gz, x, T, __ldg(f.nH + id), fa->c);
            if (ns >= 0) {
                f.N1[id] = N; f.Gx1[id] = gx; f.Gy1[id] = gy; f.Gz1[id] = gz;
                f.x[id] = x; f.T[id] = T;
                nsub_extra += ns - 1;
                nsub_max = max(nsub_max, ns);
                ncell++;
            } else if (INLINE64) {          // stiff, small grid: the fp64 redo of step_stiff_kernel, here
                double Nd = f.N1[id], gxd = f.Gx1[id], gyd = f.Gy1[id], gzd = f.Gz1[id], xd = f.x[id], Td = f.T[id];
                if (f.fix_inject && ((__ldg(f.src_bits + ((unsigned)id >> 5)) >> (id & 31)) & 1u)) Nd += source_lookup_d(f, id, fa->cd.dt);
                const int n64s = chemistry_f64<FLAGS>(Nd, gxd, gyd, gzd, xd, Td, (double)__ldg(f.nH + id), fa->cd);
                f.N1[id] = (float)Nd; f.Gx1[id] = (float)gxd; f.Gy1[id] = (float)gyd; f.Gz1[id] = (float)gzd;
                f.x[id] = (float)xd; f.T[id] = (float)Td;
                nsub_extra += n64s - 1;
                nsub_max = max(nsub_max, n64s);
                ncell++;
                n64++;
            } else {                        // stiff: the cell keeps its values; step_stiff_kernel redoes it in fp64
                const unsigned slot = atomicAdd(f.stiff_n, 1u);
                if (slot < f.stiff_cap) {
                    f.stiff_q[slot] = id;
                } else {                    // queue full (more than ncell / 16 stiff cells): this one stays fp32
                    N = f.N1[id]; gx = f.Gx1[id]; gy = f.Gy1[id]; gz = f.Gz1[id]; x = f.x[id]; T = f.T[id];
                    if (f.fix_inject && ((__ldg(f.src_bits + ((unsigned)id >> 5)) >> (id & 31)) & 1u)) N += source_lookup(f, id, fa->c.dt);
                    const int n32 = chemistry<FLAGS, false>(N, gx, gy, gz, x, T, __ldg(f.nH + id), fa->c);
                    f.N1[id] = N; f.Gx1[id] = gx; f.Gy1[id] = gy; f.Gz1[id] = gz;
                    f.x[id] = x; f.T[id] = T;
                    nsub_extra += n32 - 1;
                    nsub_max = max(nsub_max, n32);
                    ncell++;
                }
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) { qn = 0; qhead = 0; }
        __syncthreads();
    };
    // the mask is scanned in groups of FIXUP_GROUP chunks of FIXUP_THREADS words: all the group's words are loaded at
    // once and an empty group (almost all of them away from fronts and sources) costs one block-wide vote
    const int end = word0 + nwords;
    const int ngroups = (nwords + FIXUP_GROUP * FIXUP_THREADS - 1) / (FIXUP_GROUP * FIXUP_THREADS);
    // groups are handed out by a global cursor (f.stiff_n[2]): sources and fronts cluster, a static split leaves some
    // blocks with several times the cells of others
    __shared__ int s_grp;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_grp = (int)atomicAdd(f.stiff_n + 2, 1u);
        __syncthreads();
        const int grp = s_grp;
        if (grp >= ngroups) break;
        unsigned bits[FIXUP_GROUP];
        unsigned any = 0u;
#pragma unroll
        for (int k = 0; k < FIXUP_GROUP; k++) {
            const int w = word0 + (grp * FIXUP_GROUP + k) * FIXUP_THREADS + threadIdx.x;
            bits[k] = w < end ? f.defer_mask[w] : 0u;
            any |= bits[k];
        }
        if (!__syncthreads_or(any != 0u)) continue;       // (the barrier at the loop top orders s_grp's next write)
#pragma unroll
        for (int k = 0; k < FIXUP_GROUP; k++) {
            bool full = false;
            if (bits[k]) {
                const int w = word0 + (grp * FIXUP_GROUP + k) * FIXUP_THREADS + threadIdx.x;
                f.defer_mask[w] = 0u;
                unsigned bb = bits[k];
                int pos = atomicAdd(&qn, __popc(bb));
                full = pos + __popc(bb) >= FIXUP_QTHRESH;
                while (bb) {
                    const int b = __ffs(bb) - 1;
                    bb &= bb - 1;
                    queue[pos++] = w * 32 + b;
                }
            }
            // the queue's final length is the largest pos + popc any thread saw: the vote decides for the whole block.
            // (Reading qn after a plain barrier would race with the next chunk's atomicAdd of a faster thread: part of
            // the block would drain and the rest would not.)
            if (__syncthreads_or(full)) drain();
        }
    }
    __syncthreads();
    if (qn > 0) drain();
    // statistics: warp reduce, one atomic set per warp that saw work
    for (int o = 16; o > 0; o >>= 1) {
        nsub_extra += __shfl_xor_sync(0xffffffffu, nsub_extra, o);
        ncell += __shfl_xor_sync(0xffffffffu, ncell, o);
        n64 += __shfl_xor_sync(0xffffffffu, n64, o);
        nsub_max = max(nsub_max, __shfl_xor_sync(0xffffffffu, nsub_max, o));
    }
    if ((threadIdx.x & 31) == 0 && ncell > 0) {
        atomicAdd(f.stats, (unsigned long long)nsub_extra);
        atomicMax(f.stats + 1, (unsigned long long)nsub_max);
        atomicAdd(f.stats + 2, (unsigned long long)ncell);
        if (n64 > 0) atomicAdd(f.stats + 3, (unsigned long long)n64);
    }
    // the last block to finish re-arms the group cursor ([3] counts finished blocks)
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(f.stiff_n + 3, 1u) == gridDim.x - 1) { f.stiff_n[2] = 0u; f.stiff_n[3] = 0u; }
    }
}

// cells [cell0, cell1) (whole planes; for the fallback grids the whole grid): mask words [cell0 / 32, ceil(cell1 / 32))
template <int FLAGS, int GROUP, bool INLINE64>
cudaError_t launch_step_fixup_g(const FixArgs *fa, int word0, int nwords, cudaStream_t stream) {
    const int ngroups = (nwords + GROUP * FIXUP_THREADS - 1) / (GROUP * FIXUP_THREADS);
    const int blocks = ngroups < 148 * 8 ? (ngroups > 0 ? ngroups : 1) : 148 * 8;
    step_fixup_kernel<FLAGS, GROUP, INLINE64><<<blocks, FIXUP_THREADS, 0, stream>>>(fa, word0, nwords);
    return cudaGetLastError();
}

// grids of at most this many cells redo their stiff cells inside step_fixup_kernel (no step_stiff_kernel launch)
constexpr long FIXUP_INLINE64_CELLS = 1L << 21;

template <int FLAGS>
cudaError_t launch_step_fixup(const FixArgs *fa, long cell0, long cell1, bool inline64, cudaStream_t stream) {
    const int word0 = (int)(cell0 / 32), nwords = (int)((cell1 + 31) / 32) - word0;
    const int chunks = (nwords + FIXUP_THREADS - 1) / FIXUP_THREADS;
    if (inline64) return launch_step_fixup_g<FLAGS, 1, true>(fa, word0, nwords, stream);
    if (chunks >= 8 * 148 * 8) return launch_step_fixup_g<FLAGS, 8, false>(fa, word0, nwords, stream);   // >= 512^3
    if (chunks >= 2 * 148 * 8) return launch_step_fixup_g<FLAGS, 2, false>(fa, word0, nwords, stream);
    return launch_step_fixup_g<FLAGS, 1, false>(fa, word0, nwords, stream);
}

template <int FLAGS>
cudaError_t launch_step_stiff(const FixArgs *fa, cudaStream_t stream) {
    // wide enough that a few hundred thousand stiff cells get a thread each: the kernel then lasts as long as its
    // slowest cell (tens of fp64 sub-cycles), not as long as a queue of them.  (Fewer blocks on small grids change nothing:
    // its 17 us floor with nothing queued is not the chain of per-block atomics.)
    step_stiff_kernel<FLAGS><<<148 * 8, 128, 0, stream>>>(fa);
    return cudaGetLastError();
}

}  // namespace aton
