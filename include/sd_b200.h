/*
 * sd_b200.h -- C ABI of libsd_b200.so: Stokesian-dynamics mobility product on NVIDIA B200.
 *
 * The library evaluates, on one GPU and on the fly (the 3N x 3N matrix is never stored,
 * PAPER.md:109), the hot path of Kopp & Hoefling, arXiv:1205.6333:
 *
 *   v_i = mu0 F_i + sum_{j != i} T(r_i - r_j) . F_j ,   mu0 = 1/(6 pi eta a)
 *                                                        Eq. (7a)
 *   T(r) = mu0 [ 3a/(4r) (I + rr^) + a^3/(2r^3) (I - 3 rr^) ]      Eq. (7b)
 *   r < 2a: T = mu0 [ (1 - 9r/(32a)) I + 3r/(32a) rr^ ]   (Rotne-Prager-Yamakawa overlap
 *           form; the paper is silent, BASELINE.json north_star mandates it)
 *   Oseen variant: G(r) = 1/(8 pi eta r) (I + rr^)                  Eq. (4)
 *
 * and the explicit integrators it feeds:
 *   Euler     r <- r + dt M(r) F
 *   midpoint  r_h = r + dt/2 M(r) F ;  r <- r + dt M(r_h) F         (north_star)
 *
 * Conventions for every entry point
 *  - Layout: `pos`, `force`, `vel` are contiguous [N][4] records (x, y, z, pad): the paper's
 *    float4 record.  Element type is `float` for SD_PREC_F32_KAHAN and
 *    SD_PREC_F32_PLAIN, `double` for SD_PREC_F64.  The pad lane is ignored on input and
 *    written as 0 on output.  Records must be 16-byte aligned (32 bytes for double).
 *  - Unless the name ends in `_host`, data pointers are DEVICE pointers owned by the caller.
 *    The context owns every scratch buffer (packed particle records, partial sums, midpoint
 *    positions, position low words), allocated by sd_create and by the setters that change the
 *    kernel variant.  Two lazily allocated exceptions, both on first use and never inside a
 *    stream capture: the device staging of sd_mobility_apply_host (3 N records) and the cell
 *    grid of the lubrication step above 4096 particles.  Nothing else is allocated by
 *    sd_mobility_apply / sd_step / sd_lubrication_apply.
 *  - Calls must be made with the CUDA device the context was created on as the current device
 *    (SD_ERR_INVALID_ARG otherwise).  After a setter failed with SD_ERR_ALLOC / SD_ERR_CUDA the
 *    context refuses work until a setter succeeds again; its settings are kept.
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls only enqueue
 *    work; they do not synchronise the host, except sd_create, sd_destroy and the `_host`
 *    variants (which return after their result has landed in host memory).
 *  - Every function returns SD_OK or an error code; sd_last_error() gives the message of the
 *    last failure on that context (or of the last failed sd_create when ctx is NULL).
 *    Non-finite particle DATA is not checked (as in the paper's kernels).
 *  - There is no CPU fallback: without a CUDA device of compute capability 10.x sd_create
 *    fails with SD_ERR_UNSUPPORTED.
 *  - Coincident centres (r = 0, j != i): RPY contributes mu0 F_j, Oseen contributes 0.
 */
#ifndef SD_B200_H
#define SD_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sd_ctx sd_ctx; /* opaque */

typedef enum {
    SD_OK = 0,
    SD_ERR_INVALID_ARG = 1,
    SD_ERR_ALLOC = 2,
    SD_ERR_CUDA = 3,
    SD_ERR_UNSUPPORTED = 4
} sd_status;

typedef enum {
    SD_TENSOR_RPY = 0,  /* Eq. (7b) for r >= 2a, overlap form for r < 2a (default) */
    SD_TENSOR_OSEEN = 1 /* Eq. (4), unregularised, for every r > 0 */
} sd_tensor;

typedef enum {
    SD_PREC_F32_KAHAN = 0, /* fp32 terms, compensated accumulation; default */
    SD_PREC_F64 = 1,       /* fp64 terms and sums.  1/r is a 22-bit MUFU.RSQ seed on the fp32 copy of r^2
                            * plus one Newton step in fp64: relative error <= 8.6e-14 per pair (not
                            * correctly rounded; 1e-11 on the row sums is the tested bound), and r^2
                            * must lie in the fp32 range (|r| between 1e-19 and 1e19) */
    SD_PREC_F32_PLAIN = 2  /* fp32 terms, plain fp32 accumulation: ablation of PAPER.md:253-263 */
} sd_precision;

typedef enum { SD_INT_EULER = 0, SD_INT_MIDPOINT = 1 } sd_integrator;

/* Force callback for sd_step: must ENQUEUE on `stream` work that fills force[N][4] (device,
 * element type of the context's precision) from pos[N][4] (device); must not synchronise.
 * Return 0 on success; any other value aborts sd_step with SD_ERR_INVALID_ARG. */
typedef int (*sd_force_fn)(const void* pos, void* force, long long N, void* user, void* stream);

/* Create a context for N >= 1 spheres of radius a > 0 in a fluid of viscosity eta > 0 on the
 * current CUDA device.  Allocates all scratch.  Defaults: SD_TENSOR_RPY, SD_PREC_F32_KAHAN. */
sd_status sd_create(sd_ctx** out, long long N, double a, double eta);

/* Select the pair tensor / the arithmetic.  Changing the precision changes the element type
 * expected of pos/force/vel, resets the position compensation and zeroes the velocities of the
 * last product; every other setter keeps them (the lubrication correction reads them). */
sd_status sd_set_tensor(sd_ctx* ctx, sd_tensor tensor);
sd_status sd_set_precision(sd_ctx* ctx, sd_precision precision);

/* Boundary conditions (footnote 1: "a simulation box with periodic boundaries and
 * include only hydrodynamic interactions from the nearest image of each particle").
 * box_side = 0 (default): free space.  box_side = L > 0: periodic cube of side L; every
 * component of d = r_i - r_j is replaced by d - L n, n the integer nearest to d / L, before the
 * pair tensor is evaluated; the self pair stays excluded.  Positions need not lie inside the box
 * and sd_step never wraps them.  n is taken in the arithmetic of the context's precision as
 * rint(d * fl(1/fl(L))) with the product exact and ties to even (fl = rounding to float in the
 * F32 modes, to double in F64), so a pair within rounding of |d| = L/2 may see the opposite,
 * equally near image.  |d| / L must stay below 2^22 (F32) / 2^51 (F64). */
sd_status sd_set_box(sd_ctx* ctx, double box_side);

/* Step 3 of the paper's loop (Eq. 7a): vel = M(pos) force.
 * pos, force: in; vel: out (must not alias pos or force). */
sd_status sd_mobility_apply(sd_ctx* ctx, const void* pos, const void* force, void* vel,
                            void* stream);

/* Same product with HOST buffers: copies pos/force to the device, runs the product, copies
 * vel back and waits for it.  Pinned host memory makes the copies asynchronous. */
sd_status sd_mobility_apply_host(sd_ctx* ctx, const void* pos_host, const void* force_host,
                                 void* vel_host, void* stream);

/* The same product (Eq. 1 with Eq. 4 / 7; fp32 with compensated summation, free
 * space) for callers that cannot allocate device memory -- code under stream capture, tight
 * serving loops, harnesses that forbid cudaMalloc: no context, no cudaMalloc / cudaFree / allocating
 * library call, ever.  pos[N][4], force[N][4] (in) and vel[N][4] (out; must not alias the inputs)
 * are 16-byte-aligned device arrays of float on the CURRENT device; N <= sd_noalloc_max_particles()
 * = 16384, SD_ERR_UNSUPPORTED with a message (sd_last_error(NULL)) beyond that.  Two launches are
 * enqueued on `stream` (a set-up kernel and the warp-split pair kernel of sd_mobility_apply); the
 * host is not synchronised.  Scratch (partial sums of i-blocks shared by several CTAs, their ticket
 * counters and schedule, pad records) lives in ONE static device array of 4 MiB that every GPU
 * holds from the moment the library is loaded until the process exits.  Every call shares that
 * array and finds the previous call's contents in it; the set-up kernel rewrites what must start
 * clean.  Calls that overlap on the GPU (different streams, different host threads) RACE on it:
 * serialise them on one stream.  The first call on a device looks up the array's device address and
 * sets a kernel attribute (no allocation; make that call outside a stream capture).  Results agree
 * with sd_mobility_apply(PREC_F32_KAHAN) to the tolerance of that path (1e-5 relative per row). */
sd_status sd_mobility_apply_noalloc(long long N, double a, double eta, sd_tensor tensor, const void* pos,
                                    const void* force, void* vel, void* stream);
long long sd_noalloc_max_particles(void);

/* n_steps >= 0 explicit steps of size dt, pos updated in place (steps 1-3).
 * Forces, in order of precedence:
 *   fn != NULL     -> fn(pos, ctx-owned force buffer, N, user, stream) before every product;
 *   force != NULL  -> constant per-particle forces force[N][4] (device);
 *   otherwise      -> the same constant force gravity[3] on every particle.
 * Positions are carried with a context-owned low word (double-single) in
 * the fp32 modes; it stays valid while the caller does not modify pos between calls (see
 * sd_reset_compensation).  After the call sd_get_velocity returns the velocities of the last
 * product evaluated (Euler: M(r_n)F; midpoint: M(r_h)F).
 * Launch-bound loops (constant forces, no callback, 32 steps or more, N <= 32768 or the
 * lubrication correction on) are enqueued as replays of a CUDA graph of 16 steps, captured once
 * per (pos, force, gravity, dt, integrator) on a context-owned stream, plus a direct tail; the
 * kernels and therefore the results are those of step-by-step launches. */
sd_status sd_step(sd_ctx* ctx, void* pos, sd_force_fn fn, void* user, const void* force,
                  const double gravity[3], double dt, long long n_steps,
                  sd_integrator integrator, void* stream);

/* Lubrication correction.  Eq. (8), rotational terms ignored as in the paper:
 *   mu0 f_sing(r_ij) = [1/(4s) - (9/40) ln s] rr^ - (1/6) ln s (I - rr^),   s = r_ij / a - 2,
 *   force_out[i] = F_i^ext - sum'_j f_sing(r_ij) . (v_i - v_j)            (step 2)
 * the primed sum running over j != i with r_ij < 3a ("we truncate ad hoc at s = 1").  s is clamped
 * from below at 1e-3 (Eq. 8 diverges at contact and is undefined for overlapping spheres; the
 * paper never lets spheres touch); coincident centres contribute nothing.  F^ext is f_ext[N][4]
 * or, when f_ext is NULL, the uniform force gravity[3] (NULL: zero).  pos, vel, f_ext, force_out
 * are device arrays of the context's element type; force_out may be f_ext, not pos or vel.  The
 * neighbour search tests all pairs in one launch up to 1024 particles and uses a cell grid
 * rebuilt on every call above that (up to 4096 particles in the shared memory of the one kernel
 * that does the whole step; beyond that in context-owned global arrays, allocated on first use);
 * results do not depend on thread scheduling.  With sd_set_box the nearest image is used and the
 * box side must exceed 6a (9a for the cell grid, i.e. above 4096 particles), SD_ERR_UNSUPPORTED
 * otherwise.  The cut-off is decided in the context's arithmetic, the accepted pairs are
 * evaluated in fp64. */
sd_status sd_lubrication_apply(sd_ctx* ctx, const void* pos, const void* vel, const void* f_ext,
                               const double gravity[3], void* force_out, void* stream);

/* on != 0: sd_step runs the paper's full loop: before every product the forces
 * (gravity / force / the callback's) are corrected by sd_lubrication_apply with the velocities of
 * the product evaluated last (zero after sd_create; see sd_set_velocity).  Default off. */
sd_status sd_set_lubrication(sd_ctx* ctx, int on);

/* Set the "velocities of the previous step" the next lubrication correction uses: vel[N][4]
 * (device), or NULL for zero. */
sd_status sd_set_velocity(sd_ctx* ctx, const void* vel, void* stream);

/* Copy the velocities of the last product into vel_out[N][4] (device). */
sd_status sd_get_velocity(sd_ctx* ctx, void* vel_out, void* stream);

/* Forget the position low words (call after editing pos between sd_step calls). */
sd_status sd_reset_compensation(sd_ctx* ctx, void* stream);

/* Accessors. */
long long sd_num_particles(const sd_ctx* ctx);
double sd_self_mobility(const sd_ctx* ctx); /* mu0 = 1/(6 pi eta a) */
double sd_box(const sd_ctx* ctx);           /* side of the periodic cube, 0 in free space */

const char* sd_last_error(const sd_ctx* ctx);
void sd_destroy(sd_ctx* ctx);

/* =====================================================================================
 * Diagnostics, ablations and tuning knobs.  NOT needed to use the library: the calls above are
 * the product ABI.  What follows serves the tests, bench.py and the paper's
 * ablation experiments; defaults are the measured optima.
 * ===================================================================================== */

/* The static work schedule of the tiled kernels, as a pure host function (no GPU needed; the
 * library builds its own schedules with the same code).  The (i-block, j-tile) units u = b T + t,
 * B = ceil(N / particles_per_block) blocks x T = ceil(N / tile_j) tiles, are cut into
 * G = min(B T, max_ctas) contiguous pieces of equal size +-1: piece g owns units
 * [cta_u0[g], cta_u0[g+1]).  Block b collects the partial sums of pieces blk_first[b] ...
 * blk_first[b] + blk_nslots[b] - 1.  CTA x works on piece cta_piece[x]; the CTAs x, x + num_sms,
 * x + 2 num_sms, ... (which share an SM) own consecutive pieces.  dims receives {B, T, G,
 * max slots per block}; the arrays (host; sizes G+1, G, B, B) may be NULL, call once with NULL
 * arrays to learn the sizes. */
sd_status sd_schedule_plan(long long N, int particles_per_block, int tile_j, long long max_ctas,
                           int num_sms, long long* cta_u0, int* cta_piece, int* blk_first,
                           int* blk_nslots, int* dims);

/* Dispatch knobs of the small-N path (below a few thousand particles the device is
 * under-filled), for ablations and tests; the defaults are the measured crossovers.
 *   small_apply_max     : N up to which one product is ONE launch of the warp-per-particle kernel
 *                         (no pack / partial sums / finalize); < 0 restores the default (fp32 modes:
 *                         4736 in free space, 2304 in the periodic box and with sd_set_jsplit(ctx, 2);
 *                         fp64: 1000; the warp-split kernels take over there; 2560 with
 *                         sd_set_jsplit(ctx, 1)).
 *   particles_per_thread: 2, 4 or 8 particles i per thread in the tiled kernels (fp64: half of
 *                         it); 0 = automatic (by N).
 * Reallocates the scratch buffers; synchronises the device. */
sd_status sd_set_dispatch(sd_ctx* ctx, long long small_apply_max, int particles_per_thread);

/* How the j sum of one particle is split (north_star: "splits j across warps"), fp32 modes, above
 * the small-N path:
 *   mode 0  automatic: the warp-split one-launch kernel up to a measured N, the classic kernels above
 *   mode 1  classic only: the 8 warps of a CTA own different particles and share every j tile; j is
 *           split across CTAs; pack / pair / finalize kernels
 *   mode 2  warp-split wherever it exists: the 8 warps of a CTA own the same 256 particles and take
 *           an eighth of the CTA's j range each (their own bulk-copy pipelines), sums combined
 *           through shared memory, the last CTA of an i-block finishes its rows: one launch
 * Reallocates the scratch buffers; synchronises the device. */
sd_status sd_set_jsplit(sd_ctx* ctx, int mode);

/* Ablation of the memory-access schemes the paper compares (PAPER.md:111-241 and Appendix A): how
 * the j records reach the threads of the tiled kernel.
 *   0  bulk asynchronous copies into a ring of shared-memory tiles (default, the product path)
 *   1  "naive" (Alg. 1): every thread loads each record from global memory, one address per warp
 *   2  "tiling" (Alg. 2): the block copies a tile into shared memory between two barriers
 * Modes 1 and 2 exist for SD_TENSOR_RPY + SD_PREC_F32_KAHAN in free space only; otherwise, and
 * for any later change away from that combination, SD_ERR_UNSUPPORTED is returned and the context
 * is left unchanged.  Results are bit-identical across modes. */
sd_status sd_set_staging(sd_ctx* ctx, int mode);

/* Ablation of PAPER.md:253-263 ("single or double-single precision for ... (b) positions in the
 * Euler integration"): on = 1 (default) carries positions as (hi, lo) float pairs in the fp32
 * modes; on = 0 keeps them in plain fp32, r <- fl32(r + h v), low words held at zero.  No effect
 * in SD_PREC_F64.  The accumulation of the velocities, (a) in the paper, is selected by
 * sd_set_precision (SD_PREC_F32_KAHAN / SD_PREC_F32_PLAIN). */
sd_status sd_set_position_compensation(sd_ctx* ctx, int on);

/* Number of kernel launches enqueued by this context since creation (bench bookkeeping). */
long long sd_launch_count(const sd_ctx* ctx);

/* Per-kernel timing for the roofline report: while enabled, every launch of the pair kernel is
 * bracketed by CUDA events on the launching stream.  sd_profile_read waits for the recorded
 * launches, returns their summed duration [ms] and count, and clears the record.  At most 4096
 * launches are kept between reads (later ones are not recorded). */
sd_status sd_profile_enable(sd_ctx* ctx, int on);
sd_status sd_profile_read(sd_ctx* ctx, double* pair_kernel_ms, long long* pair_kernel_launches);

/* Name of the pair kernel the dispatcher picks for the current settings, e.g.
 * "pairs_f32x2_i8_rpy"; static storage. */
const char* sd_kernel_name(const sd_ctx* ctx);

/* Device micro-benchmark used to calibrate the ALU roofline: runs a dependent-chain FMA
 * kernel (fp32 packed FFMA2 when precision is an F32 mode, DFMA for SD_PREC_F64) on every SM
 * and writes the achieved TFLOP/s (FMA = 2 flop).  Synchronises the stream. */
sd_status sd_fma_peak_probe(sd_ctx* ctx, sd_precision precision, double* tflops_out,
                            void* stream);

/* The paper's Appendix A on this GPU: minimal O(N^2) memory-access kernels,
 * N threads in blocks of 128, thread j accumulates N array elements (sum of the floats of every
 * element it visits, starting from its own element in[j]) and stores the sum in out[j] (float).
 *   elem_floats  1 (float) or 4 (float4)
 *   pattern      0 linear k -> k, 1 strided k -> 131 k mod N, 2 unordered k -> (131 k + 32 j) mod N
 *   scheme       0 naive (Alg. 3), 1 small-tiling (first warp stages 32 elements, Alg. 4),
 *                2 tiling (the block stages 128 elements), 3 bulk asynchronous copies into a
 *                shared-memory ring (linear pattern only; N % 4 == 0 for float)
 * Runs one warm-up launch and `reps` timed launches on `stream`, waits for them and returns the
 * mean time per launch.  in: device array of N elements (16-byte aligned), out: N floats.  No
 * context is needed; errors are reported through sd_last_error(NULL). */
sd_status sd_access_bench(int elem_floats, int pattern, int scheme, long long N, int reps,
                          const void* in, void* out, double* ms_per_launch, void* stream);


#ifdef __cplusplus
}
#endif
#endif /* SD_B200_H */
