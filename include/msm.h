/* include/msm.h -- C ABI of libmsm_b200: the multilevel summation method (MSM) with B-spline
 * interpolation for point charges (arxiv 2510.05961, "msmJAX"; PAPER.md cited as P:<line>) as
 * hand-written CUDA for sm_100a.
 *
 * One evaluation computes, for N point charges in an orthorhombic box with full, mixed (two
 * periodic axes) or no periodicity, the MSM approximation of
 *     U = 1/2 sum_i sum_{j != i} q_i q_j / r_ij                               (Eq. 1, k(r) = 1/r)
 * together with forces -grad_i U, potentials dU/dq_i (the "charge gradient", Eq. 18) and the
 * virial -dU/d eps (the stress of P:31 times the volume, sign flipped).  Coulomb constant 1
 * (P:300).  The stages behind msm_evaluate are the paper's: short-range pair sum of k_0 with the
 * self term (Eq. 5), anterpolation (Eq. 9, Alg. 1), restriction / prolongation
 * (Eq. 19), per-level stencil convolution (Eq. 11; stencils P:268 Eq. 20 from the
 * splitting P:276 Eq. 21), the top level, and interpolation with its derivatives (P:220-230
 * Eq. 16-18).  Where PAPER.md is silent the readings of DESIGN.md apply (K1, K2, G1-G4, J1, Q,
 * T1-T4, V).
 *
 * No torch types cross this boundary: plain pointers (host or device, as stated) and sizes.
 * Nothing here throws or aborts; every call returns msm_status_t.  There is no CPU fallback: a
 * call fails with MSM_ERR_CUDA if no CUDA device is usable.
 */
#ifndef MSM_B200_H
#define MSM_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct msm_plan msm_plan_t; /* opaque; owns all device and host scratch buffers */
typedef struct msm_batch msm_batch_t; /* opaque; B plans of one geometry + the graph that runs them together */

typedef enum {
  MSM_OK = 0,
  MSM_ERR_INVALID_ARG = 1,        /* non-positive box/h/a, odd or unsupported p, levels < 1, NULL */
  MSM_ERR_UNSUPPORTED = 2,        /* exactly one periodic axis (reading T4); top grid larger than
                                     MSM_MAX_TOP_POINTS; stencil too wide for the shared memory */
  MSM_ERR_CUTOFF_TOO_LARGE = 3,   /* periodic axis with a > box/2: minimum image invalid */
  MSM_ERR_TOO_MANY_PARTICLES = 4, /* n > max_particles */
  MSM_ERR_OUT_OF_BOX = 5,         /* open-axis coordinate outside [0, box], or non-finite input */
  MSM_ERR_NOMEM = 6,
  MSM_ERR_CUDA = 7,
  MSM_ERR_SCRATCH_LIMIT = 8       /* msm_restrict_noalloc: grids need more than MSM_NOALLOC_SCRATCH_BYTES */
} msm_status_t;

typedef enum { MSM_FP64 = 0, MSM_FP32 = 1 } msm_precision_t;

#define MSM_MAX_LEVELS 32
#define MSM_MAX_TOP_POINTS 4096

/* The paper's statement of the problem (cutoff, spacing, order; cell; periodicity). */
typedef struct {
  double box[3];     /* orthorhombic edge lengths; the box is [0,box_x) x [0,box_y) x [0,box_z)   */
  int periodic[3];   /* per axis: 1 periodic, 0 open                                             */
  double h;          /* target finest grid spacing h_1.  Periodic axes use M_1 = 2^round(log2(box/h))
                        points (reading G1); open axes use h exactly              */
  double a;          /* level-zero cutoff r_cut^(0) (Eq. 3)                                 */
  int p;             /* B-spline order (support in grid cells; degree p-1): 4, 6 or 8      */
  int levels;        /* open box: number of grid levels L (the last is summed densely, untruncated
                        k_L).  Periodic / mixed: number of grids run as tiled stages; the rest of
                        the hierarchy, down to one point per periodic axis, is folded into
                        one dense operator at plan time; the result does not depend on it (G4)   */
  int precision;     /* msm_precision_t: element type of ALL particle and grid arrays            */
  int mu;            /* extra quasi-interpolation terms in omega' (reading Q); < 0: default 4     */
  int max_particles; /* capacity; msm_evaluate with n above it fails                             */
  int device;        /* CUDA device ordinal                                                      */
} msm_params_t;

typedef struct {
  int L_full;                        /* number of grid levels of the method              */
  int n_tiled;                       /* levels run as tiled stages; level n_tiled is the top grid */
  int mu;                            /* omega' setting in use                                    */
  int omega_halfwidth;               /* p/2 - 1 + mu                                             */
  int grid_dims[MSM_MAX_LEVELS][3];  /* points per axis, levels 1..L_full at index l-1            */
  int grid_lo[MSM_MAX_LEVELS][3];    /* node index of the first point (0 on periodic axes)       */
  double grid_h[MSM_MAX_LEVELS][3];  /* spacing per axis                                         */
  int stencil_taps[MSM_MAX_LEVELS];  /* taps of the sampled stencil inside the cutoff ellipsoid  */
  int pair_cells[3];                 /* short-range cell grid                                    */
  int top_points;                    /* points of the top grid (size of the dense operator)      */
  size_t device_bytes;               /* device memory owned by the plan                          */
} msm_plan_info_t;

/* Build a plan: all host-side mathematics in fp64 (grid hierarchy, two-scale mask J, quasi-
 * interpolation sequence omega', sampled stencils of every k_l and of their strain derivatives,
 * the dense top-level operator, cell-list geometry) and every device buffer for up to
 * max_particles.  On failure *plan_out is NULL. */
msm_status_t msm_plan_create(const msm_params_t *params, msm_plan_t **plan_out);

msm_status_t msm_plan_info(const msm_plan_t *plan, msm_plan_info_t *info_out);

/* Dynamic cell (with a dynamic cell the kernel stencils are recomputed from the current
 * cell; what a plan fixes is the NUMBER of grid points, the spacings follow the cell).
 * msm_plan_create_dynamic builds a plan whose stencil tables, halos and pair cells leave room for
 * every periodic box edge to shrink by up to the fraction `reserve` (0 <= reserve <= 0.5; growth
 * needs no room); msm_plan_create is the same with reserve 0. msm_plan_set_box then moves the plan
 * to new box edges without reallocating anything: the sampled stencils s_l and their strain
 * derivatives of every tiled level are recomputed ON THE DEVICE (one thread per stored tap; every
 * intermediate level has the same functional form), the cell-list and grid geometry are
 * updated, and the dense operator of the top grid (<= 4096 points) is rebuilt on the host and
 * uploaded. Open axes must keep their length (their node set follows box / h, reading G2):
 * MSM_ERR_UNSUPPORTED otherwise, and also when a periodic edge shrinks below the reserve;
 * MSM_ERR_CUTOFF_TOO_LARGE when a > box / 2. The call synchronises the device. Results afterwards
 * equal those of a plan created at the new box (up to rounding order). */
msm_status_t msm_plan_create_dynamic(const msm_params_t *params, double reserve, msm_plan_t **plan_out);
msm_status_t msm_plan_set_box(msm_plan_t *plan, const double *box /* 3 doubles */);

/* One evaluation, enqueued on cuda_stream (a cudaStream_t; NULL = the default stream).
 *   d_positions  device, n x 3 row-major (x,y,z per particle), plan precision; not modified.
 *                Periodic coordinates are wrapped into the box; open coordinates must lie in
 *                [0, box] (else MSM_ERR_OUT_OF_BOX, reported after the call completes).
 *   d_charges    device, n, plan precision; not modified.
 *   d_forces     device, n x 3, plan precision, caller order; may be NULL.
 *   d_potentials device, n, dU/dq_i, so that U = 1/2 sum q_i potentials_i; may be NULL.
 *   h_energy     host, 1 double; may be NULL.
 *   h_virial     host, 6 doubles xx yy zz xy xz yz of -dU/d eps_ab (number of grid points and a
 *                fixed, reading V); may be NULL (the strain-derivative work is then skipped).
 * The caller owns all six buffers; the plan owns every scratch buffer and msm_evaluate allocates
 * nothing. The work is stream-ordered: it starts after everything already enqueued on cuda_stream,
 * and work enqueued on cuda_stream afterwards sees d_forces / d_potentials. If h_energy or
 * h_virial is non-NULL the call waits for the evaluation and fills them (and reports
 * MSM_ERR_OUT_OF_BOX); if both are NULL it returns as soon as the work is enqueued, without any
 * host synchronisation (msm_get_results waits and reports later). A plan has one set of scratch
 * buffers: a second evaluation, on whatever stream, is ordered on the device behind the first.
 * From the second consecutive call with identical arguments on, the launch sequence is captured
 * into a CUDA graph and replayed on a plan-owned stream that is forked from and joined back into
 * cuda_stream (a small system is otherwise bound by its ~40-60 dependent kernel launches); results
 * are bit-identical either way. The short-range pair kernel runs on a second plan-owned stream
 * beside the grid pipeline and joins before the interpolation (not while per-stage profiling is
 * on).
 * Neutrality is assumed on periodic axes: the single-point top level contributes zero (reading
 * T2), which for a non-neutral input is the neutralising-background convention.
 *
 * Environment knobs, read once at msm_plan_create (debugging and measurement only; none changes a
 * result beyond rounding order): MSM_NO_GRAPH=1 (no CUDA-graph replay), MSM_NO_OVERLAP=1 (every
 * kernel on the caller's stream), MSM_GRID_STREAM_MIN=<points> (finest-grid size from which the
 * one-sweep restriction / prolongation / filter kernels run; default 4 Mi points for restriction
 * and filter, 0 for prolongation), MSM_FILTER_STREAM_MIN=<points> (the same for the filter alone),
 * MSM_CONV_SLICES=<n> / MSM_CONV_VSLICES=<n> (input-plane slices per convolution / virial tile),
 * MSM_CONV_NO_LISTS=1 (convolution kernels with the row/chunk loops instead of the entry lists),
 * MSM_TOP_BESIDE=0 (small jobs: the top-level operator after the convolution instead of beside it), MSM_CONV_GLOBAL_TAPS=1 (fp32
 * convolution reads its stencil tables from global memory), MSM_ANTERP_TILED=0 /
 * MSM_ANTERP_MIN_TILES=<n> (choice between the tiled and the gather anterpolation),
 * MSM_PAIR_SUBBINS_LOG2=<0..3> (x sub-bins per pair cell). */
msm_status_t msm_evaluate(msm_plan_t *plan, int n, const void *d_positions, const void *d_charges,
                          void *d_forces, void *d_potentials, double *h_energy, double *h_virial,
                          void *cuda_stream);

/* msm_evaluate without host outputs: enqueue only, never synchronises. want_virial != 0 also runs
 * the strain-derivative work (its result is read with msm_get_results). */
msm_status_t msm_evaluate_async(msm_plan_t *plan, int n, const void *d_positions, const void *d_charges,
                                void *d_forces, void *d_potentials, int want_virial, void *cuda_stream);

/* Wait for the plan's last evaluation and return its energy (1 double) and virial (6 doubles,
 * zeros if it was not requested); either pointer may be NULL. Returns MSM_ERR_OUT_OF_BOX if that
 * evaluation saw a coordinate outside an open axis or a non-finite input. */
msm_status_t msm_get_results(msm_plan_t *plan, double *h_energy, double *h_virial);

/* The same call with HOST buffers (the end-to-end path): copies positions and charges to plan-
 * owned device staging, evaluates, copies forces and potentials back. Pointers are host memory
 * (pinned memory makes the copies asynchronous). */
msm_status_t msm_evaluate_host(msm_plan_t *plan, int n, const void *h_positions,
                               const void *h_charges, void *h_forces, void *h_potentials,
                               double *h_energy, double *h_virial, void *cuda_stream);

/* Per-stage CUDA-event timing of the following msm_evaluate calls (off by default; when on, the
 * stages run back to back on one stream with an event between them). */
msm_status_t msm_set_profiling(msm_plan_t *plan, int enabled);

/* Stage names and milliseconds of the last profiled evaluate. The arrays belong to the plan. */
msm_status_t msm_get_stage_times(const msm_plan_t *plan, int *n_stages, const char *const **names,
                                 const float **milliseconds);

/* Number of kernels the last msm_evaluate launched (counted at the launch sites). */
msm_status_t msm_get_launch_count(const msm_plan_t *plan, int *count);

/* Parity taps: copy a grid of the last evaluate to the host as doubles, indexed [z][y][x].
 * kind 0: grid charge Q^l, 1: potential E^l (after prolongation), for 1 <= level <= n_tiled. */
msm_status_t msm_debug_copy_grid(const msm_plan_t *plan, int level, int kind, double *h_out,
                                 size_t capacity);

void msm_plan_destroy(msm_plan_t *plan);

/* Batched evaluation of `batch` independent small systems that share one geometry (box,
 * periodicity, h, a, p, levels, precision): the paper's batching of structures with fixed grid
 * counts and zero-charge padding, for the regime where one small system is dominated
 * by a constant overhead. Every system gets its own scratch buffers; the launch sequences
 * of all systems are captured as parallel branches of one CUDA graph and run side by side.
 *   h_n           host, batch ints: particles of each system (<= params->max_particles)
 *   d_positions   device, [batch][max_particles][3]; d_charges device, [batch][max_particles]:
 *                 system b uses the first h_n[b] entries of its slot (the rest is padding)
 *   d_forces / d_potentials  device, same layout, may be NULL
 *   h_energy      host, batch doubles; h_virial host, batch x 6 doubles; either may be NULL. With
 *                 both NULL the call is stream-ordered and does not synchronise.
 * The graph is rebuilt when any argument changes. Results equal msm_evaluate's for each system up
 * to rounding (a plan inside a batch sums the anterpolation of a small grid in another order). */
msm_status_t msm_batch_create(const msm_params_t *params, int batch, msm_batch_t **batch_out);
msm_status_t msm_evaluate_batch(msm_batch_t *batch, const int *h_n, const void *d_positions,
                                const void *d_charges, void *d_forces, void *d_potentials,
                                double *h_energy, double *h_virial, void *cuda_stream);
void msm_batch_destroy(msm_batch_t *batch);

/* Restriction without any allocation, for callers that cannot call cudaMalloc (code under CUDA-graph
 * capture, tight serving loops, harnesses that forbid it): coarse = I_l^{l+1} fine, the separable
 * two-scale restriction of P:258 Eq. 19 line 1 (one axis at a time; mask J_n = 2^(1-p)
 * binom(p, n + p/2), reading J1), i.e. what a plan computes between its levels l and l + 1, with
 * the two intermediate arrays of the axis passes in a file-scope device array of
 * MSM_NOALLOC_SCRATCH_BYTES (16 MiB, held by every GPU that loads the library until the process
 * exits) instead of plan-owned buffers. No plan is needed.
 *   device       CUDA device ordinal that owns d_fine and d_coarse
 *   precision    msm_precision_t: element type of both grids
 *   p            B-spline order: 4, 6 or 8
 *   fine_dims / fine_lo / coarse_dims / coarse_lo   host, 3 ints each (x, y, z): points per axis and
 *                node index of the first point, as msm_plan_info reports them for two consecutive
 *                levels (lo = 0 and coarse = fine / 2 on periodic axes; a periodic axis already at
 *                one point stays at one point)
 *   periodic     host, 3 ints
 *   d_fine       device, fine grid indexed [z][y][x]; not modified
 *   d_coarse     device, coarse grid indexed [z][y][x]; written in full
 * The caller owns both grids. The work is enqueued on cuda_stream and the call does not
 * synchronise. Needs coarse_x * fine_y * fine_z + coarse_x * coarse_y * fine_z elements of scratch
 * (the first term rounded up to 256 bytes): a larger problem returns MSM_ERR_SCRATCH_LIMIT and
 * nothing is launched (a periodic 128^3 fp64 fine grid needs 12 MiB and fits; 256^3 does not).
 * ALL calls on a device share the one array: calls that overlap on the GPU (different streams with
 * no ordering between them) race; calls on one stream are safe. The array keeps the previous call's
 * contents; nothing relies on it, every pass overwrites what the next one reads. */
#define MSM_NOALLOC_SCRATCH_BYTES (16u << 20)
msm_status_t msm_restrict_noalloc(int device, int precision, int p, const int *fine_dims,
                                  const int *fine_lo, const int *coarse_dims, const int *coarse_lo,
                                  const int *periodic, const void *d_fine, void *d_coarse,
                                  void *cuda_stream);

const char *msm_status_string(msm_status_t s);

/* Microbenchmarks used for the roofline denominators the driver does not provide (FP32 / FP64
 * FMA peak of the CUDA cores).  kind 0: FFMA, 1: DFMA, 2: FFMA2 (packed fma.rn.f32x2).  Returns TFLOP/s (2 flops per FMA) through
 * *tflops, timed with CUDA events on the given device. */
msm_status_t msm_measure_fma_peak(int device, int kind, double *tflops);

#ifdef __cplusplus
}
#endif
#endif /* MSM_B200_H */
