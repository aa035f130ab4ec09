// Internal: the context behind aton_t and the helpers the .cu files of the library share.  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/aton.h"
#include "aton_fixup.cuh"

namespace aton {
constexpr double K_BOLTZ = 1.380649e-16, EV_ERG = 1.602176634e-12, E0_EV = 13.6;
constexpr int REDUCE_BLOCKS = 148 * 8;
constexpr int N_STATS = 4;
struct SlabComm;     // aton_slab.cu: NCCL communicator, second stream and events of an overlapped slab run
}  // namespace aton

struct aton_ctx {
    aton::Grid g{};
    size_t ncell = 0;                      // cells this context advances (the slab's own planes)
    size_t nalloc = 0, plane = 0, off = 0; // allocated cells per array (slab: + 2 ghost planes), nx*ny, first own cell
    bool slab = false;                     // aton_init_slab: planes [z_begin, z_begin + nz_local) of a global grid
    int z_begin = 0, nz_local = 0, nz_global = 0;
    bool mean_set = false;                 // aton_set_mean_density overrides <n_H> of aton_set_fields
    double dx = 0, c = 0;
    aton_params_t p{};
    cudaStream_t stream = nullptr;
    float *rad[2][4] = {{nullptr, nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr, nullptr}};
    float *x = nullptr, *T = nullptr, *nH = nullptr;
    int cur = 0;
    unsigned *src_mask = nullptr;
    int *src_cell = nullptr;
    float *src_rho = nullptr;
    double *src_rho_d = nullptr;
    int n_src = 0;
    int device = 0;                        // the device current at aton_init; every entry point runs there
    unsigned long long *stats = nullptr;   // device [4]
    unsigned *defer_mask = nullptr;        // device, 1 bit per cell (variant 2)
    unsigned *src_bits = nullptr;          // device, 1 bit per cell: the cell holds a source (variant 4)
    int *stiff_q = nullptr;                // device [stiff_cap]: ids of the cells to redo in fp64 (variant 4)
    unsigned *stiff_n = nullptr;           // device [2]
    unsigned stiff_cap = 0;
    aton::FixArgs *fixargs = nullptr;            // device [2]: what the cold paths of variant 4 read, per ping-pong parity
    bool fix_dirty = true;                 // fixargs must be rewritten (dt, sources, <n_H> or buffers changed)
    double fix_dt = -1.0;
    long long fast_subcycles = 0;          // variant 2: one sub-cycle per cell and step, counted on the host
    double *partials = nullptr;            // device [REDUCE_BLOCKS+1][R_COUNT]
    double nH_mean = 1.0;
    bool have_fields = false;
    long long steps_done = 0, launches = 0;
    double time_s = 0;
    int variant = 5, tile_y = 0, tile_z = 0;
    bool timing = false;                   // aton_set_timing: CUDA events around the kernels of a step
    std::vector<cudaEvent_t> ev;           // pairs (start, stop), one pair per timed launch of the dominant step kernel
    std::vector<cudaEvent_t> ev_fix;       // the same for step_fixup_kernel ...
    std::vector<cudaEvent_t> ev_stiff;     // ... and for step_stiff_kernel
    aton::StepConst sc{};                  // constants of the step size fix_dt (prepare_step)
    aton::StepConstD scd{};
    cudaGraphExec_t step_graph = nullptr;  // two steps (one ping-pong pair) captured once for small, launch-bound grids
    bool graph_failed = false;             // capture or instantiation failed once: plain launches from then on
    long long graph_launches = 0, graph_fast = 0;   // what one replay adds to `launches` / `fast_subcycles`
    aton::SlabComm *comm = nullptr;        // aton_comm_init (slab contexts only)
    bool halo_valid = false;               // the ghost planes of the current buffer hold the neighbours' boundary planes
    char err[512] = "";
};

namespace aton {

extern char g_init_error[512];

inline int fail(aton_ctx *ctx, int code, const char *fmt, ...) {
    char *dst = ctx ? ctx->err : g_init_error;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

#define CU(ctx, call)                                                                         \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? ATON_ENOMEM : ATON_ECUDA,      \
                        "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

// shared between the .cu files (defined in aton_api.cu)
int check_dt(aton_ctx *ctx, double *dt, const char *who);                    // dt <= 0 -> Courant 0.8; ATON_EINVAL if unstable
cudaError_t prepare_step(aton_ctx *ctx, double dt);                          // step constants + the cold paths' arguments
cudaError_t launch_step_planes(aton_ctx *ctx, int zb, int ze);               // one step of planes [zb, ze) of the current buffer
int run_reduce(aton_ctx *ctx, bool full, double *host_out);                  // two-pass reduction -> host_out[R_COUNT]
void sums_from_reduce(aton_ctx *ctx, const double *r, const unsigned long long *st, double *sums);
void diag_from_sums(const aton_ctx *ctx, const double *sums, aton_diag_t *out);
void slab_comm_free(aton_ctx *ctx);                                          // aton_slab.cu

}  // namespace aton
