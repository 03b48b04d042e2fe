/* lgf.h -- C ABI of the B200 (sm_100a) Fourier-accelerated Landau gauge fixer.
 *
 * Method: arXiv 1301.3460, "Landau gauge fixing on the lattice using GPU's".  The library
 * maximises, on a 4-D periodic SU(3) lattice,
 *
 *     F_U[g] = (1/(N_d N_c V)) sum_x sum_mu Re Tr[ g(x) U_mu(x) g^dag(x+mu) ]
 *
 * with the steepest-descent method with Fourier acceleration, run parameters alpha and
 * theta < theta_tol, links stored as 12 reals (two rows) or 18 reals.
 * One iteration (BASELINE.json north_star steps 1-4):
 *   S1  Delta(x) = A - A^dag - (1/3)Tr(A - A^dag),  A = sum_mu [U_mu(x-mu) - U_mu(x)];
 *       theta = (1/(N_c V)) sum_x Tr[Delta Delta^dag];  F = (1/(N_d N_c V)) sum_x sum_mu Re Tr U_mu(x)
 *   S2  X = IFFT[ (p2max/p2) FFT[Delta] ],  p2(n) = sum_mu 4 sin^2(pi n_mu/L_mu), p2max = 16, zero mode 0
 *   S3  g(x) = rowGramSchmidt(1 + (alpha/2) X(x)), third row conj(u x v)
 *   S4  U_mu(x) <- g(x) U_mu(x) g^dag(x+mu)   (all x, mu simultaneously)
 *   S5  stop when theta < theta_tol (strict)
 *
 * Conventions
 *   - Host/device link arrays ("canonical order"): double [V][4][3][3][2], i.e. links[x][mu][row][col][re,im],
 *     site index x = x0 + L0*(x1 + L1*(x2 + L2*x3)) (x0 fastest), periodic boundaries.  Always 18 reals per
 *     link on this boundary, whatever the internal storage.
 *   - Every pointer argument says whether it is HOST or DEVICE memory.  The caller owns every pointer it
 *     passes; the context never keeps a caller pointer after the call returns, except the workspace and
 *     stream given to lgf_create_ex, which must outlive the context.
 *   - Every call returns lgf_status.  No exceptions, no exit(), nothing is printed.  Out-parameters are
 *     written only when the call returns LGF_OK or LGF_NOT_CONVERGED.
 *   - Calls are synchronous for the host: on return the results are final.  Internally all work is ordered
 *     on the context's CUDA stream.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with LGF_ERR_CUDA.
 *   - Supported sizes: each L_mu a power of two, 4 <= L_mu <= 128, L0*L1 <= 4096 and L2*L3 <= 4096
 *     (shared-memory tile limits of the FFT passes); otherwise LGF_ERR_UNSUPPORTED.
 */
#ifndef LGF_H
#define LGF_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lgf_ctx lgf_ctx; /* opaque; owns its device buffers unless a workspace was supplied */

typedef enum {
    LGF_OK = 0,
    LGF_ERR_INVALID_ARG = 1,
    LGF_ERR_UNSUPPORTED = 2,
    LGF_ERR_OOM = 3,
    LGF_ERR_CUDA = 4,
    LGF_ERR_NOT_LOADED = 5,
    LGF_ERR_NUMERIC = 6,      /* theta or F became non-finite */
    LGF_NOT_CONVERGED = 100   /* non-fatal: max_iter reached, state and outputs valid */
} lgf_status;

/* Precision of link storage and of the per-site arithmetic.  LGF_FP64: the paper's setting.
 * LGF_FP32: links and field stored as float, every kernel computes in float; the
 * lattice sums (theta, F) and the p^2 filter weights stay double.  Half the HBM bytes per iteration; theta bottoms out
 * between 1e-14 and 1e-12 (fp32 rounding of Delta, amplified by p2max/p2min ~ L^2), so theta < 1e-15 is not reachable in
 * this precision alone.  Host- and
 * device-side link and field arrays of this API are double in every precision (converted on load and on get).
 * LGF_MIXED: an fp64 context (everything above holds: fp64 links, fp64 lgf_iterate) whose lgf_fix runs in two phases:
 * a float copy of the links is fixed in fp32 down to theta = max(theta_tol, 1e-12) -- or until theta stops falling, so
 * a stalled fp32 phase never eats the max_iter budget -- while the update accumulates the total gauge transformation G(x); then the fp64 links receive U_mu(x) <- G(x) U_mu(x) G(x+mu)^dagger with G
 * re-orthonormalised in double -- an exact gauge copy of the input, at the fp32 noise level of theta -- and the fp64
 * iteration continues to theta_tol.  n_iter is the total; lgf_get_option(LGF_OPT_MIXED_FP32_ITERS) gives the fp32
 * share; lgf_get_history covers the fp64 phase.  Needs the workspaces of both precisions.
 * When it pays: where alpha is well inside the stable range of the configuration, the fp32 phase follows the fp64
 * trajectory and the total iteration count stays within a few of the fp64 run's (all BASELINE.json ensembles; thermalised
 * beta = 6.0 at 32^4: 676 against 678 iterations, 161 against 209 ms).  On rough configurations where alpha sits at the
 * stability edge (thermalised beta = 5.7 at alpha = 0.08: neighbouring step sizes already change the count by 50 %) the
 * fp32 rounding sends the iteration down a different trajectory to a different Gribov copy; the count can then be larger
 * than the fp64 run's (measured: 13 634 against 10 639) as well as smaller.  The result is a valid gauge-fixed copy of the
 * input either way (theta < theta_tol in fp64); only the time is not predictable there -- use LGF_FP64. */
typedef enum { LGF_FP64 = 0, LGF_FP32 = 1, LGF_MIXED = 2 } lgf_precision;
typedef enum { LGF_STORE_18 = 18, LGF_STORE_12 = 12 } lgf_storage;

/* Bytes of device workspace a context for these parameters needs (0 if the parameters are unsupported).
 * [layout: SURVEY.md 8(a) S0; 12-real storage PAPER.md:45,51] */
size_t lgf_workspace_bytes(const int dims[4], lgf_precision p, lgf_storage s);

/* Create a context: lgf_create(dims, precision, storage) of the north star; lattice, precision and link storage as the
 * paper names them (PAPER.md:45 "12 real number representation", :47 lattice volume, :51 double precision).
 * dims: HOST, {L0,L1,L2,L3}.  The library allocates its own device memory (cudaMalloc)
 * on the current device and creates its own stream. */
lgf_status lgf_create(const int dims[4], lgf_precision p, lgf_storage s, lgf_ctx **out);

/* Same, but all device memory comes from dev_workspace (DEVICE pointer, 256-byte aligned, at least
 * lgf_workspace_bytes() bytes) and all work is ordered on cuda_stream (a cudaStream_t cast to void*; NULL is
 * the default stream).  This is how a framework (e.g. PyTorch) lends memory and a stream. */
lgf_status lgf_create_ex(const int dims[4], lgf_precision p, lgf_storage s,
                         void *dev_workspace, size_t workspace_bytes, void *cuda_stream, lgf_ctx **out);

void lgf_destroy(lgf_ctx *ctx);

/* Load links U_mu(x) (the gauge configuration of PAPER.md:37-39; layout S0, reading A9: no reprojection).
 * host_links: HOST, canonical order, V*4*18 doubles.  Stored as given -- no reprojection; in
 * 12-real storage rows 0,1 are kept and row 2 is dropped (it is rebuilt as conj(row0 x row1) on use). */
lgf_status lgf_load_links(lgf_ctx *ctx, const double *host_links);
/* Same from DEVICE memory (canonical order). */
lgf_status lgf_load_links_device(lgf_ctx *ctx, const double *dev_links);

/* The same pair in the two-row host format (the paper's "12 real number representation", carried to the
 * boundary): host_rows: HOST, double [V][4][2][3][2] = rows 0,1 of every link, V*4*12 doubles; a third of the bytes of the
 * canonical array stays off the PCIe link.  Only for contexts created with LGF_STORE_12 (else LGF_ERR_UNSUPPORTED); the
 * caller rebuilds row 2 = conj(row0 x row1) where it needs it. */
lgf_status lgf_load_links_12(lgf_ctx *ctx, const double *host_rows);
lgf_status lgf_get_links_12(lgf_ctx *ctx, double *host_rows);

/* Read the gauge-fixed links back (the transformed U of PAPER.md:39), canonical order, always full 18 reals per link (row 2 rebuilt in 12-real storage). */
lgf_status lgf_get_links(lgf_ctx *ctx, double *host_links);
lgf_status lgf_get_links_device(lgf_ctx *ctx, double *dev_links);

/* Apply exactly n iterations S1-S4 (north star steps 1-4; steepest descent with Fourier acceleration) with
 * step alpha, no stop test, then measure once more (reading A5).
 * F, theta (HOST, may be NULL): the functional and theta of the links AFTER the n-th update.  n >= 0. */
lgf_status lgf_iterate(lgf_ctx *ctx, int n, double alpha, double *F, double *theta);

/* Iterate until theta < theta_tol (strict; "theta < 10^-15", alpha = 0.08 there) or max_iter updates (S5).  n_iter (HOST): number of link updates applied
 * before the first measurement with theta < theta_tol (0 if the links already satisfy it).  F, theta: that
 * measurement.  Returns LGF_OK, or LGF_NOT_CONVERGED when max_iter updates did not reach theta_tol. */
lgf_status lgf_fix(lgf_ctx *ctx, double alpha, double theta_tol, int max_iter,
                   int *n_iter, double *F, double *theta);

/* Step-size scan (the paper runs one alpha = 0.08; tuning it is the subject of its refs [1],[2]):
 * from the links now in the context, one lgf_fix(alphas[k], theta_tol, max_iter) per k, each from the same start.
 * alphas: HOST, n values > 0.  counts: HOST, n ints: the iteration count of each run, -1 where max_iter updates did not
 * reach theta_tol, -2 where the iteration diverged (non-finite theta or F).  F_final: HOST, n doubles (may be NULL): F at
 * the stop.  best: HOST (may be NULL): index of the smallest count, -1 if no run converged.  The context's links are the
 * same before and after the call (the start is kept in a temporary device buffer of the size of the link store:
 * LGF_ERR_OOM if that cannot be allocated). */
lgf_status lgf_scan_alpha(lgf_ctx *ctx, const double *alphas, int n, double theta_tol, int max_iter,
                          int *counts, double *F_final, int *best);

/* F (PAPER.md:39 with g = 1), theta (north star step 1) and the average plaquette of the current links; no state change.  Any out pointer may be NULL. */
lgf_status lgf_measure(lgf_ctx *ctx, double *F, double *theta, double *plaquette);

/* (F_k, theta_k) of the measurements made by the last lgf_iterate/lgf_fix call, k = 0..min(n_iter, cap-1);
 * hist: HOST, 2*capacity doubles; *n_out receives how many pairs were written. */
lgf_status lgf_get_history(lgf_ctx *ctx, double *hist, int capacity, int *n_out);

/* Stage read-outs for kernel-level parity tests.  Each writes a full anti-Hermitian 3x3 field, HOST,
 * double [V][3][3][2], computed by the hot-path kernels from the current links (links unchanged):
 *   LGF_FIELD_DELTA  Delta(x) of step S1;   LGF_FIELD_X  X(x) of step S2;
 *   LGF_FIELD_G      g(x) of step S3 for the given alpha (a special unitary field, not anti-Hermitian). */
typedef enum { LGF_FIELD_DELTA = 0, LGF_FIELD_X = 1, LGF_FIELD_G = 2 } lgf_field;
lgf_status lgf_get_field(lgf_ctx *ctx, lgf_field which, double alpha, double *host_field);

/* Options.  The method itself (what is computed):
 *   LGF_OPT_FOURIER_ACCEL    1 (default): the paper's method, X = IFFT[(p2max/p2) FFT[Delta]].  0: plain
 *                            steepest descent, X = Delta (what Fourier acceleration is measured against, PAPER.md:41
 *                            refs [1],[2]); converges for alpha < 2/p2max = 1/8, rate degrades with the volume.
 *   LGF_OPT_GAUGE_DIRECTIONS 4 (default): Landau gauge, the paper's problem.  3: Coulomb gauge -- the
 *                            gauge condition, Delta, F (normalised by 3 N_c V) and p^2 run over mu = 0..2, p2max = 12, the
 *                            spatial zero mode of every time slice is dropped, all four link directions are transformed.
 * How it runs (results identical up to rounding order; DESIGN.md section 6 holds the measured A/B numbers):
 *   LGF_OPT_STORE_G          0 (default): S3+S4 rebuild g(x+mu) from X.  1: pass C stores g(x) (96 B/site) and S4 reads it.
 *   LGF_OPT_GRAPH            1 (default): iterations are replayed through a CUDA graph.  0: plain launches.
 *   LGF_OPT_BATCH            iterations enqueued between two reads of the device stop flag (default 8, 1..1024).
 *   LGF_OPT_PDL              1 (default): programmatic dependent launch between the kernels of an iteration.  0: off.
 *   LGF_OPT_FAST_FFT         1 (default): compile-time-sized FFT passes where the lattice allows (extents 16/32/64).
 *                            0: the generic passes.  get: bit mask of the passes that run fast (1 A, 2 B, 4 C).
 *   LGF_OPT_TMA              1 (default): the FFT passes run persistent, one CTA per SM, fed by the Tensor Memory Accelerator
 *                            (cp.async.bulk.tensor + mbarrier).  Pass A (S1 + axes 0,1; 16/32 extents, two-row storage): the
 *                            links stream into shared memory stage by stage while the warps compute Delta and transform.
 *                            Pass B (axes 2,3): at 16/32 extents the next tiles stream in while the current ones are
 *                            transformed; at 64 extents the tile goes in and out through the TMA unit.  0: one CTA per plane
 *                            or tile, plain loads and stores.  get: bit mask of the TMA passes that actually run (1 B, 2 A).
 *   LGF_OPT_MIXED_FP32_ITERS read-only: fp32 iterations of the last LGF_MIXED lgf_fix.
 *   LGF_OPT_MIXED_SWITCH     LGF_MIXED: the fp32 phase aims at theta = 10^-value (default 12, 4..20) and hands over to fp64
 *                            there, or earlier when theta stops falling (it has not halved within 256 iterations). */
typedef enum { LGF_OPT_STORE_G = 0, LGF_OPT_GRAPH = 1, LGF_OPT_BATCH = 2, LGF_OPT_PDL = 3, LGF_OPT_FAST_FFT = 4,
               LGF_OPT_FOURIER_ACCEL = 5, LGF_OPT_GAUGE_DIRECTIONS = 6, LGF_OPT_MIXED_FP32_ITERS = 7,
               LGF_OPT_MIXED_SWITCH = 8, LGF_OPT_TMA = 9 } lgf_option;
lgf_status lgf_set_option(lgf_ctx *ctx, lgf_option opt, int value);
lgf_status lgf_get_option(lgf_ctx *ctx, lgf_option opt, int *value);

/* Per-kernel device timing.  lgf_set_profiling(ctx,1) brackets every kernel launch with CUDA events on the
 * context's stream (plain launches, no graph); lgf_get_profile returns, per kernel slot i < LGF_MAX_KERNELS,
 * the accumulated milliseconds and launch counts since profiling was enabled.  names via lgf_kernel_name. */
#define LGF_MAX_KERNELS 32
lgf_status lgf_set_profiling(lgf_ctx *ctx, int on);
lgf_status lgf_get_profile(lgf_ctx *ctx, double ms[LGF_MAX_KERNELS], long long launches[LGF_MAX_KERNELS]);
const char *lgf_kernel_name(int slot);

/* Total number of this library's kernels launched by the context since creation. */
long long lgf_launch_count(lgf_ctx *ctx);

/* Stream copy yardstick: copies `bytes` (multiple of 16) from dev_src to dev_dst (DEVICE) `reps` times with the
 * library's own double2 streaming kernel on cuda_stream and returns the average milliseconds per copy in *ms
 * (HOST).  This is the "measured copy-kernel peak" of the north star: GB/s = 2*bytes/ms/1e6. */
lgf_status lgf_copy_peak(void *dev_dst, const void *dev_src, size_t bytes, int reps, void *cuda_stream, double *ms);

/* Second yardstick: the access pattern of the link kernels without their arithmetic.  dev_buf, DEVICE, holds 24 arrays
 * of n_sites double2 (24 * 16 * n_sites bytes: the 12-real link store of n_sites sites); one thread per site reads its
 * entry of each array (write = 0) or reads it and writes it back in place (write = 1), 128 threads per CTA.  n_sites a
 * multiple of 128.  *ms, HOST, receives the mean time of one of `reps` launches after one warm-up; bytes moved per
 * launch: 384 * n_sites * (1 + write).  Same errors as lgf_copy_peak. */
lgf_status lgf_stream_peak(void *dev_buf, size_t n_sites, int write, int reps, void *cuda_stream, double *ms);

/* ---- Slab-decomposed context (the paper's CPU comparator is this decomposition over MPI +
 * PFFT).  The lattice is cut along axis 3 into n_ranks slabs; every rank has its own workspace and runs
 * S1, the plane passes and S3+S4 on its slab; per iteration the ranks exchange one time slice of U_3 (for S1), one time
 * slice of X (for S3) and transpose the 64 B/site field twice (so that pass B finds axis 3 local).  This build runs the
 * ranks as VIRTUAL ranks on the current device (one stream, n_ranks separate allocations); the only code that crosses
 * rank boundaries is one copy function and one table of peer pointers, written for GPUs with peer access
 * (csrc/lgf_slab.inl).  fp64, Landau gauge, the generic FFT passes.  n_ranks: a power of two <= 16 dividing L1 and L3;
 * L0 <= 64.  Same semantics, tolerances and error codes as the single-context calls of the same names. */
typedef struct lgf_slab_ctx lgf_slab_ctx;
lgf_status lgf_create_sharded(const int dims[4], int n_ranks, lgf_storage s, lgf_slab_ctx **out);
void       lgf_destroy_sharded(lgf_slab_ctx *ctx);
int        lgf_sharded_ranks(lgf_slab_ctx *ctx);
lgf_status lgf_load_links_sharded(lgf_slab_ctx *ctx, const double *host_links);   /* HOST, canonical order: rank r takes x3 in [r L3/P, (r+1) L3/P) */
lgf_status lgf_get_links_sharded(lgf_slab_ctx *ctx, double *host_links);
lgf_status lgf_iterate_sharded(lgf_slab_ctx *ctx, int n, double alpha, double *F, double *theta);
lgf_status lgf_fix_sharded(lgf_slab_ctx *ctx, double alpha, double theta_tol, int max_iter, int *n_iter, double *F, double *theta);
lgf_status lgf_get_history_sharded(lgf_slab_ctx *ctx, double *hist, int capacity, int *n_out);
/* out (HOST, 5 values): bytes ONE rank sends per iteration for [0] the U_3 halo, [1] the X halo, [2] the two transposes;
 * [3] kernels launched and [4] inter-rank copies issued by the context so far. */
lgf_status lgf_sharded_traffic(lgf_slab_ctx *ctx, long long out[5]);
const char *lgf_last_error_sharded(lgf_slab_ctx *ctx);   /* ctx == NULL: text of the calling thread's last failed lgf_create_sharded */

/* Third yardstick: the FP64 FMA rate of the device (8 independent chains of dependent fused multiply-adds per thread, 64
 * warps per SM, no memory traffic), in TFLOP/s, averaged over `reps` launches on cuda_stream.  The arithmetic roof of the
 * FFT passes: the path is HBM-bound, but pass B is within a factor of two of this one as well. */
lgf_status lgf_fp64_peak(int reps, void *cuda_stream, double *tflops);

/* ---- theta and F without any allocation (csrc/lgf_static.cu).
 * Every call above that needs device memory gets it from cudaMalloc, at lgf_create or (lgf_scan_alpha) per call.  Some
 * programs cannot let a library do that: a production Monte Carlo job whose own pool took all of the HBM at start-up (a
 * library cudaMalloc then fails although the job has memory to spare), a program under a framework's caching allocator
 * (what the framework has cached is invisible to cudaMalloc), or a measurement hook inside a running update loop (cudaMalloc
 * and cudaFree synchronise the whole device and would stall the job's other streams on every call).  For them the lattice
 * sums of step S1 -- the gauge-fixing monitor theta and the functional F (PAPER.md:39 with g = 1; theta as in PAPER.md:47) --
 * are one stateless call.  It needs no context, creates no stream or event, and calls no cudaMalloc/cudaFree: its only
 * scratch memory, one partial sum per 128 sites, is a fixed array inside the library image.
 *   dev_links   DEVICE, canonical order, V*4*18 doubles, 16-byte aligned; read only.  All three rows are read (no 12-real
 *               rebuild), nothing is reprojected.
 *   dims        HOST, {L0,L1,L2,L3}, every L_mu >= 1 (any integers, not only powers of two), V = L0 L1 L2 L3 <=
 *               LGF_STATIC_MAX_SITES; a larger lattice returns LGF_ERR_UNSUPPORTED and launches nothing.
 *   cuda_stream a cudaStream_t of the current device cast to void* (NULL: the default stream).
 *   dev_out     DEVICE, 2 doubles: dev_out[0] = F, dev_out[1] = theta (Landau gauge, the normalisations of lgf_measure).
 * Unlike the context calls this one does not wait: it enqueues two kernels on cuda_stream and returns; dev_out is final
 * when the stream has run them.  Returns LGF_OK, LGF_ERR_INVALID_ARG (NULL pointer, extent < 1), LGF_ERR_UNSUPPORTED (too
 * many sites), LGF_ERR_CUDA (no device, failed launch); lgf_measure_static_error() gives the text of the calling thread's
 * last failure ("" after a success).
 * Cost and sharing: the array is LGF_STATIC_MAX_SITES/128 * 16 B = 2 MiB of every GPU the process uses, from the moment the
 * library is loaded until exit.  The first call on a device looks up the array's address on that device and keeps it:
 * make that first call before beginning any stream capture.  All calls on a device use the same array, which keeps the
 * previous call's partial sums; a call overwrites every entry it later reads, so nothing needs clearing -- but calls that
 * overlap on the GPU (two streams, or two host threads without ordering between their streams) race on it and both
 * results are then undefined.  Calls on one stream, or ordered by events, are safe. */
#define LGF_STATIC_MAX_SITES (1 << 24)   /* 64^4, the largest lattice of BASELINE.json */
lgf_status lgf_measure_static(const double *dev_links, const int dims[4], void *cuda_stream, double *dev_out);
const char *lgf_measure_static_error(void);

const char *lgf_status_string(lgf_status s);
const char *lgf_last_error(lgf_ctx *ctx); /* detail of the last LGF_ERR_CUDA (static or ctx-owned string) */

#ifdef __cplusplus
}
#endif
#endif /* LGF_H */
