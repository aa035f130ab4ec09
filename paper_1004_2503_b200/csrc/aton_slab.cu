// z-slab decomposition over several GPUs (the paper's multi-GPU mode: cube
// decomposition, boundary faces of (N, F) staged GPU -> host -> MPI -> host -> GPU every step, 10-15 % of the step).
// Here: slabs along z, so a halo is one contiguous nx*ny plane per field; the planes travel device to device with
// ncclSend / ncclRecv straight out of / into the field arrays (no pack, no unpack, no host staging), on a second
// stream, while the interior planes of the step are computed:
//
//   per step:  boundary planes (z = 1 and z = nz_local)  ->  event  ->  [comm stream] exchange of the NEW buffer's
//              boundary planes into the neighbours' ghost planes      ||  [main stream] interior planes 2 .. nz_local-1
//              the next step's boundary kernels wait for the exchange's event.
//
// NCCL is resolved at run time (dlopen of libnccl.so.2): the library loads and runs single-GPU without it, and a
// process that already holds torch's NCCL shares it.  The communicator is the library's own (created from a unique id
// the caller distributes), so nothing depends on the caller's framework.
#include <dlfcn.h>
#include <nccl.h>      // types and constants only; every function is called through the table below

#include "aton_ctx.cuh"

namespace aton {

struct NcclApi {
    ncclResult_t (*GetUniqueId)(ncclUniqueId *) = nullptr;
    ncclResult_t (*CommInitRank)(ncclComm_t *, int, ncclUniqueId, int) = nullptr;
    ncclResult_t (*CommDestroy)(ncclComm_t) = nullptr;
    ncclResult_t (*Send)(const void *, size_t, ncclDataType_t, int, ncclComm_t, cudaStream_t) = nullptr;
    ncclResult_t (*Recv)(void *, size_t, ncclDataType_t, int, ncclComm_t, cudaStream_t) = nullptr;
    ncclResult_t (*AllGather)(const void *, void *, size_t, ncclDataType_t, ncclComm_t, cudaStream_t) = nullptr;
    ncclResult_t (*GroupStart)() = nullptr;
    ncclResult_t (*GroupEnd)() = nullptr;
    const char *(*GetErrorString)(ncclResult_t) = nullptr;
    bool ok = false;
};

static NcclApi *nccl_api() {
    static NcclApi api;
    static bool tried = false;
    if (tried) return &api;
    tried = true;
    void *h = dlopen("libnccl.so.2", RTLD_NOW | RTLD_GLOBAL);
    if (!h) h = dlopen("libnccl.so", RTLD_NOW | RTLD_GLOBAL);
    if (!h) return &api;
#define ATON_SYM(name) *(void **)(&api.name) = dlsym(h, "nccl" #name)
    ATON_SYM(GetUniqueId); ATON_SYM(CommInitRank); ATON_SYM(CommDestroy); ATON_SYM(Send); ATON_SYM(Recv);
    ATON_SYM(AllGather); ATON_SYM(GroupStart); ATON_SYM(GroupEnd); ATON_SYM(GetErrorString);
#undef ATON_SYM
    api.ok = api.GetUniqueId && api.CommInitRank && api.CommDestroy && api.Send && api.Recv && api.AllGather &&
             api.GroupStart && api.GroupEnd && api.GetErrorString;
    return &api;
}

struct SlabComm {
    ncclComm_t comm = nullptr;          // null: a single rank that is its own neighbour (periodic wrap by device copies)
    int rank = 0, world = 1, below = 0, above = 0;
    cudaStream_t cstream = nullptr;     // the exchange runs here, beside the interior planes
    cudaEvent_t ev_boundary = nullptr, ev_halo = nullptr;
    double *d_sums = nullptr;           // device [ATON_NSUMS * (1 + world)]: all-gather of the raw diagnostic sums
};

void slab_comm_free(aton_ctx *ctx) {
    SlabComm *c = ctx->comm;
    if (!c) return;
    if (c->comm) nccl_api()->CommDestroy(c->comm);
    if (c->cstream) cudaStreamDestroy(c->cstream);
    if (c->ev_boundary) cudaEventDestroy(c->ev_boundary);
    if (c->ev_halo) cudaEventDestroy(c->ev_halo);
    cudaFree(c->d_sums);
    delete c;
    ctx->comm = nullptr;
}

#define NC(ctx, call)                                                                                      \
    do {                                                                                                   \
        ncclResult_t r_ = (call);                                                                          \
        if (r_ != ncclSuccess)                                                                             \
            return fail(ctx, ATON_ECUDA, "%s: %s (%s:%d)", #call, nccl_api()->GetErrorString(r_), __FILE__, __LINE__); \
    } while (0)

// Boundary planes of buffer `b` -> the neighbours' ghost planes of buffer `b`, enqueued on the comm stream:
// my first own plane becomes the ghost plane ABOVE the slab below, my last own plane the ghost plane BELOW the slab above.
static int exchange(aton_ctx *ctx, int b) {
    SlabComm *c = ctx->comm;
    const size_t pl = ctx->plane;
    const int nzl = ctx->nz_local;
    if (!c->comm) {      // one rank: periodic wrap inside the slab
        for (int v = 0; v < 4; v++) {
            float *a = ctx->rad[b][v];
            CU(ctx, cudaMemcpyAsync(a + (size_t)(nzl + 1) * pl, a + pl, pl * sizeof(float), cudaMemcpyDeviceToDevice, c->cstream));
            CU(ctx, cudaMemcpyAsync(a, a + (size_t)nzl * pl, pl * sizeof(float), cudaMemcpyDeviceToDevice, c->cstream));
        }
        return ATON_OK;
    }
    NcclApi *n = nccl_api();
    NC(ctx, n->GroupStart());
    for (int v = 0; v < 4; v++) {
        float *a = ctx->rad[b][v];
        // posted in the same order on every rank, so with world == 2 (both neighbours are the same peer) the first
        // send pairs with the peer's first receive
        NC(ctx, n->Send(a + pl, pl, ncclFloat, c->below, c->comm, c->cstream));
        NC(ctx, n->Recv(a + (size_t)(nzl + 1) * pl, pl, ncclFloat, c->above, c->comm, c->cstream));
        NC(ctx, n->Send(a + (size_t)nzl * pl, pl, ncclFloat, c->above, c->comm, c->cstream));
        NC(ctx, n->Recv(a, pl, ncclFloat, c->below, c->comm, c->cstream));
    }
    NC(ctx, n->GroupEnd());
    return ATON_OK;
}

// all ranks' raw sums combined (entries 0-10 and 14 add, 11-12 max, 13 min); synchronises the main stream
static int global_sums(aton_ctx *ctx, double *sums) {
    SlabComm *c = ctx->comm;
    if (!c || !c->comm) return ATON_OK;
    const int w = c->world;
    std::vector<double> all((size_t)ATON_NSUMS * w);
    CU(ctx, cudaMemcpyAsync(c->d_sums, sums, sizeof(double) * ATON_NSUMS, cudaMemcpyHostToDevice, ctx->stream));
    NC(ctx, nccl_api()->AllGather(c->d_sums, c->d_sums + ATON_NSUMS, ATON_NSUMS, ncclDouble, c->comm, ctx->stream));
    CU(ctx, cudaMemcpyAsync(all.data(), c->d_sums + ATON_NSUMS, sizeof(double) * ATON_NSUMS * w, cudaMemcpyDeviceToHost, ctx->stream));
    CU(ctx, cudaStreamSynchronize(ctx->stream));
    for (int k = 0; k < ATON_NSUMS; k++) {
        double v = all[k];
        for (int r = 1; r < w; r++) {
            const double u = all[(size_t)r * ATON_NSUMS + k];
            v = (k == 11 || k == 12) ? std::max(v, u) : (k == 13 ? std::min(v, u) : v + u);
        }
        sums[k] = v;
    }
    return ATON_OK;
}

}  // namespace aton

using namespace aton;

extern "C" {

int aton_comm_unique_id(unsigned char *id, int nbytes) {
    if (!id || nbytes != ATON_COMM_ID_BYTES) return fail(nullptr, ATON_EINVAL, "aton_comm_unique_id: nbytes must be ATON_COMM_ID_BYTES");
    static_assert(sizeof(ncclUniqueId) == ATON_COMM_ID_BYTES, "ATON_COMM_ID_BYTES must match ncclUniqueId");
    NcclApi *n = nccl_api();
    if (!n->ok) return fail(nullptr, ATON_ECUDA, "aton_comm_unique_id: libnccl.so.2 not found");
    ncclUniqueId u;
    if (n->GetUniqueId(&u) != ncclSuccess) return fail(nullptr, ATON_ECUDA, "aton_comm_unique_id: ncclGetUniqueId failed");
    std::memcpy(id, &u, sizeof(u));
    return ATON_OK;
}

int aton_comm_init(aton_t *ctx, const unsigned char *id, int nbytes, int rank, int world) {
    if (!ctx) return ATON_EINVAL;
    if (!ctx->slab) return fail(ctx, ATON_ESTATE, "aton_comm_init: not a slab context");
    if (world < 1 || rank < 0 || rank >= world) return fail(ctx, ATON_EINVAL, "aton_comm_init: need 0 <= rank < world");
    if (id && nbytes != ATON_COMM_ID_BYTES) return fail(ctx, ATON_EINVAL, "aton_comm_init: nbytes must be ATON_COMM_ID_BYTES");
    if (!id && world != 1) return fail(ctx, ATON_EINVAL, "aton_comm_init: a NULL id is only valid for world == 1");
    if (world == 1 && ctx->nz_local != ctx->nz_global)
        return fail(ctx, ATON_EINVAL, "aton_comm_init: world == 1 needs the slab to span the whole grid");
    cudaSetDevice(ctx->device);
    slab_comm_free(ctx);
    SlabComm *c = new (std::nothrow) SlabComm();
    if (!c) return fail(ctx, ATON_ENOMEM, "aton_comm_init: host allocation failed");
    ctx->comm = c;
    c->rank = rank; c->world = world;
    c->below = (rank + world - 1) % world;
    c->above = (rank + 1) % world;
    CU(ctx, cudaStreamCreateWithFlags(&c->cstream, cudaStreamNonBlocking));
    CU(ctx, cudaEventCreateWithFlags(&c->ev_boundary, cudaEventDisableTiming));
    CU(ctx, cudaEventCreateWithFlags(&c->ev_halo, cudaEventDisableTiming));
    CU(ctx, cudaMalloc((void **)&c->d_sums, sizeof(double) * ATON_NSUMS * (1 + world)));
    if (id) {
        NcclApi *n = nccl_api();
        if (!n->ok) return fail(ctx, ATON_ECUDA, "aton_comm_init: libnccl.so.2 not found");
        ncclUniqueId u;
        std::memcpy(&u, id, sizeof(u));
        NC(ctx, n->CommInitRank(&c->comm, world, u, rank));
    }
    ctx->halo_valid = false;
    return ATON_OK;
}

int aton_step_slab(aton_t *ctx, double dt, int n_steps) {
    if (!ctx) return ATON_EINVAL;
    if (!ctx->slab || !ctx->comm) return fail(ctx, ATON_ESTATE, "aton_step_slab: needs a slab context with aton_comm_init done");
    if (!ctx->have_fields) return fail(ctx, ATON_ESTATE, "aton_step_slab: call aton_set_fields first");
    if (n_steps < 0) return fail(ctx, ATON_EINVAL, "aton_step_slab: n_steps < 0");
    if (ctx->variant != 4 && ctx->variant != 5)
        return fail(ctx, ATON_ESTATE, "aton_step_slab: a slab context runs kernel variants 4 and 5 only");
    if (int rc = check_dt(ctx, &dt, "aton_step_slab")) return rc;
    cudaSetDevice(ctx->device);
    SlabComm *c = ctx->comm;
    const int nzl = ctx->nz_local;
    if (n_steps > 0) CU(ctx, prepare_step(ctx, dt));
    for (int s = 0; s < n_steps; s++) {
        if (!ctx->halo_valid) {          // first step after an upload (or after aton_step): fill the ghost planes
            CU(ctx, cudaEventRecord(c->ev_boundary, ctx->stream));
            CU(ctx, cudaStreamWaitEvent(c->cstream, c->ev_boundary, 0));
            if (int rc = exchange(ctx, ctx->cur)) return rc;
            CU(ctx, cudaEventRecord(c->ev_halo, c->cstream));
        }
        CU(ctx, cudaStreamWaitEvent(ctx->stream, c->ev_halo, 0));          // ghost planes of the current buffer are in
        // boundary planes first ...
        CU(ctx, launch_step_planes(ctx, 1, 2));
        if (nzl > 1) CU(ctx, launch_step_planes(ctx, nzl, nzl + 1));
        CU(ctx, cudaEventRecord(c->ev_boundary, ctx->stream));
        // ... their exchange (of the buffer just written) beside the interior planes
        CU(ctx, cudaStreamWaitEvent(c->cstream, c->ev_boundary, 0));
        if (int rc = exchange(ctx, 1 - ctx->cur)) return rc;
        CU(ctx, cudaEventRecord(c->ev_halo, c->cstream));
        if (nzl > 2) CU(ctx, launch_step_planes(ctx, 2, nzl));
        ctx->cur = 1 - ctx->cur;
        ctx->halo_valid = true;
        ctx->steps_done++;
        ctx->time_s += dt;
    }
    // leave the main stream ordered after the last exchange, so that any later call sees complete ghost planes
    if (n_steps > 0) CU(ctx, cudaStreamWaitEvent(ctx->stream, c->ev_halo, 0));
    return ATON_OK;
}

int aton_reduce_global(aton_t *ctx, aton_diag_t *out) {
    if (!ctx || !out) return ATON_EINVAL;
    double sums[ATON_NSUMS];
    if (int rc = aton_reduce_sums(ctx, sums, ATON_NSUMS)) return rc;
    if (int rc = global_sums(ctx, sums)) return rc;
    diag_from_sums(ctx, sums, out);
    return ATON_OK;
}

int aton_sync_mean_density(aton_t *ctx) {
    if (!ctx) return ATON_EINVAL;
    if (!ctx->have_fields) return fail(ctx, ATON_ESTATE, "aton_sync_mean_density: no fields set");
    double sums[ATON_NSUMS];
    if (int rc = aton_reduce_sums(ctx, sums, ATON_NSUMS)) return rc;
    if (int rc = global_sums(ctx, sums)) return rc;
    return aton_set_mean_density(ctx, sums[3] / sums[0]);
}

}  // extern "C"
