/*
 * aton.h -- C ABI of the B200-native ATON hot path.
 *
 * The operation is the explicit moment radiative-transfer step of Aubert & Teyssier,
 * "Reionization simulations powered by GPUs I" on a uniform periodic 3-D grid:
 *   transport of the photon density N and flux F with the M1 closure and a Lax-Friedrichs
 *   intercell flux (Eq.3-7; appendix Eq.A1-A5), then per cell the
 *   source term and the sub-cycled hydrogen photo-chemistry / cooling operator Phi of Eq.A4
 *   (Eq.13-15), in the order "transport, then the chemistry
 *   and the cooling".
 * The host only drives: fields go up once, every step runs on the GPU, fields
 * and the global means of PAPER.md:L149/L303 come back on request.
 *
 * All entry points are plain C.  No call aborts or throws; each returns ATON_OK (0) or a negative
 * code and leaves a message in aton_last_error().  Calls on one context are not thread-safe;
 * different contexts are independent.  Everything runs on the CUDA stream given to aton_init
 * (a cudaStream_t cast to void*, NULL = the legacy default stream) on the device that is current
 * at aton_init.  There is no CPU fallback: without a CUDA device aton_init returns ATON_ECUDA.
 *
 * Layout of every field: C order [nz][ny][nx], x fastest; cell (i,j,k) at i + nx*(j + ny*k);
 * float32; cubic cells dx = lx_cm/nx; periodic in x, y and z (wrapped in-kernel, no ghost layer).
 * Units are CGS: n_H, N [cm^-3]; F [photons cm^-2 s^-1]; T [K]; x = n_HII/n_H; rate [photons/s];
 * dt [s].  Pointers are host or device pointers as said by the `on_device` argument; the caller
 * owns every array it passes, the library copies and never keeps a caller pointer.
 */
#ifndef ATON_H
#define ATON_H

#ifdef __cplusplus
extern "C" {
#endif

#define ATON_OK 0
#define ATON_EINVAL (-1) /* bad argument: NULL, bad grid, unstable dt, position outside [0,1], ... */
#define ATON_ENOMEM (-2) /* device or host allocation failed */
#define ATON_ECUDA (-3)  /* CUDA error (sticky; text in aton_last_error) */
#define ATON_ESTATE (-4) /* call out of order, e.g. aton_step before aton_set_fields */

typedef struct aton_ctx aton_t; /* opaque; owned by the library, released by aton_free */

/* nx % 4 == 0 (128-bit accesses along x), ny, nz >= 1; nx*ny*nz < 2^31. */
typedef struct { int nx, ny, nz; } aton_grid_t;

/* Physical side along x in cm.  Cells are cubic: dx = lx_cm / nx. */
typedef struct { double lx_cm; } aton_box_t;

/* Units and physics switches.  Zero-initialise, then set; 0 means "default" where noted. */
typedef struct {
    double c_cm_s;       /* speed of light of the transport; 0 => 2.99792458e10 ("c full speed") */
    double sigma_n;      /* number-averaged photoionisation cross-section, cm^2 (2.93e-18) */
    double sigma_e;      /* energy-averaged cross-section, cm^2 (2.49e-18) */
    double e_photon_eV;  /* mean ionising photon energy, eV (20.27) */
    int recomb_case;     /* 1: case B (on-the-spot); 0: case A + recombination radiation */
    int cooling;         /* 0: T frozen (isothermal); 1: photo-heating + cooling, sub-cycled */
    int coll_ion;        /* collisional ionisation and its cooling on/off */
    int clump_model;     /* recombination clumping C_R of Eq.15:
                            0 none; 1: C = max(1, a + b*delta), delta = n_H/<n_H> - 1;
                            2: C = max(1, a * n_H^b) (PAPER.md:L259 power law) */
    double clump_a, clump_b;
    double redshift;     /* >= 0: Compton cooling off the CMB at this z; < 0: off */
    double eps_sub;      /* sub-cycle tolerance on the thermal energy change; 0 => 0.1 */
    int max_sub;         /* sub-cycle cap per cell and step; 0 => 16384 */
    double clump_i_a, clump_i_b; /* photon-atom cross clumping C_I of Eq.15 ("C_I ~ n_H^0.2"):
                            C_I = max(1, a * n_H^b) multiplies the photo-ionisation rate and the absorption;
                            a <= 0 => C_I = 1 (the variant the paper also ran, L269-271) */
    int flux;            /* intercell flux ("HLL or the simpler Lax-Friedrich scheme"): 0 = Lax-Friedrichs at
                            speed c (the one the paper used; the product kernel); 1 = HLL with the M1 wave speeds (tiled
                            kernels on grids with nx % 32 == 0 and ny % 8 == 0 -- packed fp32x2 where nx % 64 == 0: 2.0 x
                            the Lax-Friedrichs step --, a one-thread-per-cell kernel on the others; a slab context takes the tiled kernels only) */
} aton_params_t;

/* Global diagnostics (PAPER.md:L149 volume-weighted x, L303-305 mass-weighted, Eq.15 Gamma = c sigma_n N). */
typedef struct {
    double x_vol, x_mass;         /* <x>_V = mean x ; <x>_M = sum(n_H x)/sum(n_H) */
    double gamma_vol, gamma_mass; /* photo-ionisation rate c*sigma_n*N [1/s], volume / mass weighted */
    double photons_total;         /* sum N dx^3 */
    double T_vol;                 /* mean T */
    double f_max;                 /* max reduced flux |F|/(cN) over cells with N > 0 */
    double N_min;                 /* min N */
    double frac_x_half;           /* fraction of cells with x >= 0.5 */
    long long n_nonfinite;        /* cells holding a NaN/Inf in any of N, F, x, T */
    long long subcycles_total;    /* chemistry sub-cycles summed over cells and steps since aton_set_fields */
    long long subcycles_max;      /* largest per-cell, per-step sub-cycle count seen */
    long long cells_subcycled;    /* cell-steps redone outside the one-sub-step fast path: cells that needed more than
                                     one sub-cycle (variants 2, 4) and, for variant 4, the source cells */
    long long steps_done;         /* steps since aton_set_fields */
    double time_s;                /* sum of dt since aton_set_fields */
    long long cells_fp64;         /* of cells_subcycled: cell-steps whose sub-cycling was redone in fp64 because heating
                                     and cooling cancelled (the 10 % rule's sub-step is then ill-conditioned in fp32) */
} aton_diag_t;

/* Create a context: allocates 11 float32 device arrays of nx*ny*nz (7 fields + 4 ping-pong) and one bit
 * per cell of work flags.
 * `stream` is borrowed for the life of the context.  On failure *out is NULL. */
int aton_init(aton_t **out, const aton_grid_t *grid, const aton_box_t *box,
              const aton_params_t *params, void *cuda_stream);

/* Upload the state {n_H, x, T, N, F}.  N, Fx, Fy, Fz may each be NULL = zero
 * (dark start).  n_H must be > 0 everywhere (checked: ATON_EINVAL).  Resets the step counter, the
 * sub-cycle statistics and <n_H> of the clumping law.  Synchronises the stream. */
int aton_set_fields(aton_t *ctx, const float *nH, const float *x, const float *T, const float *N,
                    const float *Fx, const float *Fy, const float *Fz, int on_device);

/* Replace the source list (n = 0 clears it).  pos: n x 3 floats (x,y,z) in box units [0,1];
 * rate: n doubles, photons/s, >= 0.  Nearest-grid-point: cell = floor(pos*n) mod n per axis, one
 * emitter per cell, rates of sources sharing a cell are summed.  The binning, the sort by cell and the
 * fp64 merge run on the host (device arrays are copied down first): not a per-step call, 2e5 sources take milliseconds.
 * Synchronises. */
int aton_set_sources(aton_t *ctx, long long n, const float *pos, const double *rate, int on_device);

/* courant * dx / (3c): the unsplit 3-D Lax-Friedrichs step is stable for c*dt/dx <= 1/3
 * (Eq.7 L80-83 gives dt < dx/c; reading S3).  Negative on a NULL context. */
double aton_courant_dt(const aton_t *ctx, double courant);

/* Advance n_steps steps of size dt [s] (dt <= 0 => aton_courant_dt(ctx, 0.8)).  Each step:
 * transport -> source injection -> chemistry/cooling.  Asynchronous on the stream; the state at
 * t + n_steps*dt is current afterwards whatever the parity of n_steps.  ATON_EINVAL if
 * c*dt/dx > 1/3 or n_steps < 0; ATON_ESTATE before aton_set_fields. */
int aton_step(aton_t *ctx, double dt, int n_steps);

/* Download the state.  Any pointer may be NULL = skip.  Synchronises the stream. */
int aton_get_fields(aton_t *ctx, float *nH, float *x, float *T, float *N, float *Fx, float *Fy,
                    float *Fz, int on_device);

/* Global diagnostics of the current state (deterministic two-pass reduction).  Synchronises. */
int aton_reduce(aton_t *ctx, aton_diag_t *out);

/* Select the step kernel: 5 (default, the product) = row-wide warps (a warp owns a 128-cell row segment, a CTA 8 or 16
 * rows that exchange their y terms through shared memory behind one mbarrier phase per plane; needs nx % 128 == 0 and
 * ny % 8 == 0; any other grid falls through to variant 4, then 2);
 * 4 = warp-autonomous 32 x 4 (or 64 x 2) tiles, no inter-warp synchronisation (needs nx % 32 == 0 and ny % 4 == 0, or
 * nx % 64 == 0 and ny % 2 == 0; any other grid runs the variant-2 kernel).  Variants 4 and 5 flag their source cells and
 * the cells that need sub-cycling for step_fixup_kernel (stiff cells go on to the fp64 step_stiff_kernel) and give
 * bit-identical results;
 * 2 = CTA-tiled fused kernel + the same fix-up kernels (the fallback for grids the others cannot tile);
 * 0 = reference kernel (one thread per cell, neighbours from global memory; a cross-check).
 * tile_y / tile_z choose the tile shape (0 = default; variant 2: tile_y in {6, 14} rows; variant 4: tile_y 4 = 32 x 4
 * warp tiles (default), 2 = 64 x 2; variant 5: tile_y 16 (default when ny % 16 == 0) or 8 rows per CTA; tile_z = planes per z-chunk);
 * results agree between variants to rounding and do not depend on the tile shape (bitwise).  ATON_EINVAL for anything
 * else (variants 1 and 3 of round 1 are gone). */
int aton_set_kernel(aton_t *ctx, int variant, int tile_y, int tile_z);

/* Number of kernels launched by the library on this context since aton_init. */
long long aton_launch_count(const aton_t *ctx);

/* Measurement aid (bench.py's roofline): with on != 0 every later aton_step brackets the dominant
 * kernel of each step (the fused transport + injection + chemistry kernel; not the sub-cycle fix-up)
 * with CUDA events on the context's stream.  Calling it again (on or off) discards the events. */
int aton_set_timing(aton_t *ctx, int on);

/* Sum [ms] and number of the bracketed launches since aton_set_timing(ctx, 1).  Synchronises. */
int aton_kernel_time(aton_t *ctx, double *ms_total, long long *n_launches);

/* The same for the other two kernels of a step: step_fixup_kernel (the sub-cycling cells and, for variant 4, the source
 * cells) and step_stiff_kernel (the fp64 redo of the cells whose fp32 sub-cycling is not accurate enough). */
int aton_fixup_time(aton_t *ctx, double *ms_fixup, double *ms_stiff, long long *n_launches);

/* ---- slab decomposition along z (the paper's multi-GPU mode, PAPER.md:L471-484,
 * re-cut as z slabs whose one-plane halo of (N, F) is one contiguous block per field) ----
 *
 * aton_init_slab creates a context that advances planes [z_begin, z_begin + nz_local) of the GLOBAL grid
 * `global_grid` (needs a grid kernel variant 4 can tile: nx % 32 == 0 and ny % 4 == 0, or nx % 64 == 0 and ny % 2 == 0).  It holds nz_local + 2 planes per array: its
 * own planes between a ghost plane below and one above.  aton_set_fields / aton_get_fields then take arrays of
 * nz_local planes; aton_set_sources takes positions in the GLOBAL box and keeps the sources of the slab;
 * aton_reduce reports the slab's own means.  Before EVERY aton_step(ctx, dt, 1) the caller exchanges halos:
 *   aton_halo_pack(ctx, send_lo, send_hi)      own first / last plane of N, Gx, Gy, Gz -> two device buffers
 *   (send_hi goes to the slab above as its recv_lo, send_lo to the slab below as its recv_hi; periodic in z;
 *    how the buffers travel -- NCCL send/recv, peer copies -- is the caller's business)
 *   aton_halo_unpack(ctx, recv_lo, recv_hi)    two device buffers -> ghost plane below / above
 * Each buffer is [4][ny][nx] float32 on the device (fields N, Gx, Gy, Gz with G = F/c as carried internally).
 * Both calls are asynchronous on the context's stream.  A slab run is bit-identical to the undivided run. */
int aton_init_slab(aton_t **out, const aton_grid_t *global_grid, const aton_box_t *box,
                   const aton_params_t *params, void *cuda_stream, int z_begin, int nz_local);
int aton_halo_pack(aton_t *ctx, float *send_lo, float *send_hi);
int aton_halo_unpack(aton_t *ctx, const float *recv_lo, const float *recv_hi);

/* <n_H> of the linear clumping law (clump_model 1): aton_set_fields computes it over the context's own cells;
 * a slab must be given the GLOBAL mean (all-reduced by the caller) before aton_set_fields or aton_step. */
int aton_set_mean_density(aton_t *ctx, double nH_mean);

/* Raw sums of the context's own cells, to be combined across slabs (entries 0-10 and 14 add, 11-12 take the max, 13 the min):
 * [0] cells [1] sum x [2] sum n_H x [3] sum n_H [4] sum N [5] sum n_H N [6] sum T [7] cells with x >= 0.5
 * [8] non-finite cells [9] sub-cycles [10] cells redone outside the fast path [11] max f [12] max sub-cycles [13] min N
 * [14] cells redone in fp64.  n must be ATON_NSUMS.  Synchronises. */
#define ATON_NSUMS 15
int aton_reduce_sums(aton_t *ctx, double *sums, int n);

/* The diagnostics of aton_reduce formed from raw sums that the caller has combined across slabs (all the arithmetic of
 * the means -- <x>_V, <x>_M, Gamma = c sigma_n N, photons = sum N dx^3 -- stays in the library).  No device work. */
int aton_diag_from_sums(aton_t *ctx, const double *sums, int n, aton_diag_t *out);

/* <n_H> of the linear clumping law from combined raw sums: aton_set_mean_density(ctx, sums[3] / sums[0]). */
int aton_set_mean_from_sums(aton_t *ctx, const double *sums, int n);

/* ---- the same slabs with the exchange inside the library (one call per run of steps, exchange overlapped) ----
 *
 * aton_comm_unique_id: rank 0 obtains an id (ATON_COMM_ID_BYTES bytes, an ncclUniqueId) and hands it to every rank by
 * whatever means the caller has.  aton_comm_init(ctx, id, nbytes, rank, world) then creates the library's own NCCL
 * communicator over the `world` slab contexts (rank r owns the r-th slab in z order; collective: every rank calls it),
 * a second CUDA stream and the events of the overlap.  id == NULL is allowed for world == 1 (the slab spans the whole
 * grid and wraps onto itself by device copies; no NCCL needed).  libnccl.so.2 is looked up at run time.
 *
 * aton_step_slab(ctx, dt, n_steps): n steps; each step computes the slab's two boundary planes first, sends them
 * (ncclSend / ncclRecv straight out of / into the field arrays: no pack / unpack, no host staging -- the paper's
 * exchange costs 10-15 % of a step) on the second stream while the interior planes are computed, and the
 * next step's boundary kernels wait for the arrival.  Collective; asynchronous on the context's streams; bit-identical
 * to the undivided run.  aton_reduce_global all-gathers the raw sums and returns the diagnostics of the WHOLE box;
 * aton_sync_mean_density makes <n_H> of the linear clumping law the global mean (call it once after aton_set_fields). */
#define ATON_COMM_ID_BYTES 128
int aton_comm_unique_id(unsigned char *id, int nbytes);
int aton_comm_init(aton_t *ctx, const unsigned char *id, int nbytes, int rank, int world);
int aton_step_slab(aton_t *ctx, double dt, int n_steps);
int aton_reduce_global(aton_t *ctx, aton_diag_t *out);
int aton_sync_mean_density(aton_t *ctx);

/* ---- analysis and source front end around the step (nothing here runs per step) ---- */

/* Clumping-factor measurement (section 3.2.1): over every block x block x block cells of the current
 * state (the paper: 8^3 cells of its fine run = one cell of its coarse run),
 *   C_R = <n_H^2 x^2> / <n_H x>^2,   C_I = <N (1-x) n_H> / (<N> <(1-x) n_H>)      (L247),
 * with the block's mean density <n_H> and its ionised fraction <n_H x>/<n_H> (the two variables the paper bins C against,
 * Fig.12-13).  A factor whose denominator vanishes is 1.  Each output is [nz/block][ny/block][nx/block] float32, host or
 * device as said by on_device; block must divide nx, ny and nz.  Undivided contexts only.  Synchronises. */
int aton_clumping_blocks(aton_t *ctx, int block, float *nH_mean, float *x_mean, float *C_R, float *C_I, int on_device);

/* 2-D distribution of two per-cell quantities of the current state (the Gamma(n_H), x(n_H), (1-x)(n_H) planes of PAPER.md
 * Fig.5-19; L417).  A value v lands in bin floor((f(v) - lo)/(hi - lo) * nbins) of its axis, f = log10 on a log axis;
 * values outside [lo, hi) (or <= 0 on a log axis) are tallied in *outside.  counts is [nb][na] int64 (counts[ib*na + ia]),
 * host or device as said by on_device; na * nb <= 4096.  Integer counts: deterministic.  Synchronises. */
#define ATON_Q_NH 0       /* n_H [cm^-3] */
#define ATON_Q_X 1        /* ionised fraction x */
#define ATON_Q_NEUTRAL 2  /* 1 - x */
#define ATON_Q_T 3        /* T [K] */
#define ATON_Q_N 4        /* photon density N [cm^-3] */
#define ATON_Q_GAMMA 5    /* photo-ionisation rate c sigma_n N [1/s] (Eq.15) */
int aton_histogram2d(aton_t *ctx, int quantity_a, int quantity_b, int log_a, int log_b, double a_lo, double a_hi,
                     double b_lo, double b_hi, int na, int nb, long long *counts, long long *outside, int on_device);

/* Source front end (section 2.3): the star particles of snapshot p+1 -> emission rates for the transfer
 * from t_p to t_p1 [s, ages of the Universe], then aton_set_sources.  Per particle: pos (box units), age at t_p1 [s],
 * lifetime L as an ionising source [s] (the paper draws it between 5 and 20 Myr: the draw is the caller's), n_baryons;
 * Ndot = photons_per_baryon * n_baryons / L (the paper: 24 000 - 98 000 photons per stellar baryon).  With
 * a_p = age - (t_p1 - t_p): a_p > L discarded; a_p < 0 (born in the interval) the diluted rate min(age, L)/(t_p1 - t_p) Ndot;
 * otherwise min(1, (L - a_p)/(t_p1 - t_p)) Ndot -- each branch emits exactly the photons the star emits in the interval.
 * Then Eq.8-9: Ndot_eff = Ndot f_esc B, B = max(1, a_b exp(k_b / t)) at the middle of the interval (k_b in s; Table 1;
 * DESIGN.md readings G5, G6).  Arrays are host or device as said by on_device.  Synchronises. */
int aton_set_star_sources(aton_t *ctx, long long n, const float *pos, const double *age, const double *lifetime,
                          const double *nbaryons, double photons_per_baryon, double t_p, double t_p1, double f_esc,
                          double a_b, double k_b, int on_device);

/* Thomson optical depth, Eq.10: tau = c sigma_T int n_e dt for a history x(z) of the mass-weighted
 * ionised fraction (n points, z ascending, HOST arrays) in flat LCDM: n_e = x nH0 (1+z)^3, H = H0 sqrt(Om (1+z)^3 + 1 - Om)
 * [H0 in 1/s, nH0 in cm^-3]; trapezoid rule.  Synchronises. */
int aton_thomson_tau(aton_t *ctx, long long n, const double *z, const double *x, double nH0, double H0, double Om, double *tau);

/* The raw sums of aton_reduce_sums for callers that must not allocate (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): no context, no cudaMalloc / cudaFree, no synchronisation -- two kernels enqueued on
 * `cuda_stream` (a cudaStream_t cast to void*; NULL = the legacy default stream) of the CURRENT device.  The partial sums of
 * the two-pass reduction live in a static __device__ array of 104 192 bytes that every GPU holds from the moment it loads the
 * library until the process exits.
 * nH, x, T, N, Fx, Fy, Fz: DEVICE arrays of `ncell` floats each (any grid shape), 16-byte aligned; c_cm_s <= 0 => 2.99792458e10.
 * sums: DEVICE array of ATON_NOALLOC_NSUMS doubles, written when the stream reaches the call (the caller owns every array):
 *   [0] cells [1] sum x [2] sum n_H x [3] sum n_H [4] sum N [5] sum n_H N [6] sum T [7] cells with x >= 0.5
 *   [8] non-finite cells [9] max f = |F|/(cN) [10] min N [11] min n_H
 * ([0]-[8] are entries [0]-[8] of aton_reduce_sums, [9] its [11], [10] its [13]; Eq.15).
 * Limits: ncell a positive multiple of 4, at most 2^31 - 4 = 2 147 483 644 cells (ATON_EINVAL beyond, message in
 * aton_last_error(NULL)).  Every call on a device SHARES the static array, which keeps the last call's contents (nothing in it
 * has to start at zero: the rows a call reads are the rows it wrote): calls on one stream are ordered and safe, calls that
 * OVERLAP on the GPU (other streams, concurrently replayed graphs) race and give wrong sums. */
#define ATON_NOALLOC_NSUMS 12
int aton_field_sums_noalloc(const float *nH, const float *x, const float *T, const float *N, const float *Fx, const float *Fy,
                            const float *Fz, long long ncell, double c_cm_s, void *cuda_stream, double *sums);

void aton_free(aton_t *ctx);

/* Message of the last failing call on ctx (ctx-owned), or of the last failing aton_init if ctx is
 * NULL (static storage).  Never NULL. */
const char *aton_last_error(const aton_t *ctx);

#ifdef __cplusplus
}
#endif
#endif /* ATON_H */
