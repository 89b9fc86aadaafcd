/* fredopt.h -- C-ABI of the B200-native (sm_100a) hot path of FREDopt's plan optimisation.
 *
 * The library implements ONE thing: the superiorized, simultaneous (Cimmino-type) feasibility-seeking
 * iteration over the sparse spot->voxel influence matrices D (dose) and L (LET-weighted dose) of
 * "GPU-accelerated FREDopt package for simultaneous dose and LETd proton radiotherapy plan optimization via
 * superiorization methods" (arxiv 2509.20012; cited below as PAPER.md:<line>), i.e.
 *
 *   AMSrelaxDLET  (Fig. 2)  relaxed projections onto per-voxel dose / cDL half-spaces,
 *                                             then the clamp fluence_j < 0 -> 0;
 *   SuperiorDLET  (Fig. 3)  perturbations x' = x - beta * grad chi^2(x), beta = beta0*a^s,
 *                                             accepted iff chi^2 decreases, interleaved with AMS steps;
 *   chi^2         (Eq. 2,  PAPER.md:207)      sum_PTV w (Dref - D(x))^2 + sum_OAR w (cDLref - cDL(x))^2;
 *   LETd = l / d  (Eq. 1,  PAPER.md:56-64)    with the dose as denominator;
 *   plus the OAR LETd limit linearised as <L_i - LETmax * D_i, x> <= 0, the proximity function and the
 *   violation count (BASELINE.json north_star; not in the paper).
 *
 * The readings of the paper that fix every detail (simultaneous form, sign of the lower-bound branch, weight
 * normalisation, ...) are listed in DESIGN.md, "Readings of the paper".
 *
 * Conventions
 *   - rows = voxels (V = n_rows), columns = spots (S = n_cols); x in R^S is the spot-weight ("fluence") vector.
 *   - every pointer argument may be a HOST or a DEVICE pointer (detected with cudaPointerGetAttributes) unless
 *     stated otherwise; caller arrays are BORROWED for the duration of the call only; outputs are
 *     caller-allocated.  fredopt_create copies what it needs: inputs may be freed on return.
 *   - one plan = one GPU, one CUDA stream (given at creation; NULL = a stream the plan creates and owns, with
 *     cudaStreamDefault flags, i.e. ordered against the legacy default stream as any blocking stream is -- the
 *     legacy stream itself cannot be captured into a CUDA graph).  Calls enqueue on that stream; a call that writes host memory synchronises the stream before returning, a call with
 *     device outputs only does not.
 *   - arithmetic: matrix values are stored as given (fp32; as IEEE halves of their roundings with fredopt_create_options.value_bits = 16), indices as 16 bits where that is exact (n_cols <= 65536;
 *     row indices of the transposes inside 65536-row blocks) and int32 otherwise, offsets int64; every vector the
 *     iteration keeps (x, d, l, g, u, v) and every accumulator / scalar / decision is fp64 on the device.
 *     fp32 scalars cross the ABI as their bit patterns and are widened, never recomputed.
 *   - every function returns FREDOPT_OK (0) or a negative error code; no exception or abort crosses the ABI;
 *     on failure outputs and plan state are untouched (fredopt_create: *out = NULL).
 *   - requires a device of compute capability 10.x (built for sm_100a only): FREDOPT_UNSUPPORTED_ARCH otherwise.
 *     There is no CPU fallback.
 */
#ifndef FREDOPT_H
#define FREDOPT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FREDOPT_OK                 0
#define FREDOPT_INVALID_ARG       -1
#define FREDOPT_OUT_OF_MEMORY     -2
#define FREDOPT_CUDA_ERROR        -3
#define FREDOPT_UNSUPPORTED_ARCH  -4
#define FREDOPT_UNSUPPORTED       -5

typedef struct fredopt_plan fredopt_plan;   /* opaque */

/* Compressed sparse rows.  row_ptr: n_rows+1 entries, non-decreasing, row_ptr[0] = 0, row_ptr[n_rows] = nnz.
 * col_idx / values: nnz entries; within a row the columns are strictly increasing and < n_cols; values finite. */
typedef struct {
    int64_t n_rows, n_cols, nnz;
    const int64_t *row_ptr;
    const int32_t *col_idx;
    const float   *values;
} fredopt_csr;

/* Bounds of one structure (label s = 1..n_struct uses bounds[s-1]); NaN = absent.
 * Inputs of Figs. 2-3: U_D, L_D, U_cDLET, L_cDLET, w; Dref, cDLref of Eq. (2). */
typedef struct {
    float weight;               /* w_s > 0: weight / priority of the structure              */
    float dose_lo, dose_hi;     /* L_D <= <D_i, x> <= U_D                                                  */
    float dl_lo, dl_hi;         /* L_cDLET <= <L_i, x> <= U_cDLET                                          */
    float letd_max;             /* <L_i - letd_max * D_i, x> <= 0      (north_star)                        */
    float dose_ref, dl_ref;     /* Dref, cDLref of Eq. (2): cost terms w (ref - value)^2                   */
} fredopt_bounds;

/* Filled by fredopt_get_stats (synchronises). */
typedef struct {
    int64_t k;                  /* iterations done (Fig. 3's k)                                            */
    int64_t s;                  /* step-size exponent consumed so far (Fig. 3's s + 1)                     */
    int64_t trials;             /* perturbation trials evaluated so far (= s)                              */
    int64_t n_violated;         /* declared sets with a non-zero residual at the point the last AMS step   */
                                /*   of fredopt_iterate was taken from, or at the last fredopt_proximity   */
    int64_t n_sets;             /* declared constraint sets                                                */
    int64_t n_zero_norm_sets;   /* declared sets whose row has zero norm (take no part in the step)        */
    int64_t n_active_rows;      /* voxels with label != 0                                                  */
    int64_t nnz;                /* non-zeros per matrix (union pattern)                                    */
    int64_t nnz_active;         /* non-zeros in active rows                                                */
    int64_t alg_bytes_iter;     /* algorithmic bytes of ONE superiorized iteration ("Bytes")    */
    int64_t block_rows;         /* rows per stored block row of the labelled voxels (1, 2 or 4)            */
    int64_t entries_active;     /* stored entries of the labelled rows: (block row, spot) pairs of the     */
                                /*   union patterns; entries_active * block_rows >= nnz_active values      */
    double  last_beta;          /* last accepted beta (0 if none)                                          */
    double  phi;                /* chi^2 at the perturbed point of the last iteration (superiorized,       */
                                /*   simultaneous form; otherwise over the rows the last pass visited)     */
    double  prox;               /* proximity 1/2 sum w^ r^2/|a|^2 at that same point / last proximity call */
    double  weight_sum;         /* W: sum of the weights of the participating sets                         */
} fredopt_stats;

/* Options (fredopt_set_option). */
#define FREDOPT_OPT_ETA            0   /* eta of Fig. 3: lambda_k = lambda * eta^k; default 1      */
#define FREDOPT_OPT_REDUCTIONS     1   /* reductionsN of Fig. 3; default 1                         */
#define FREDOPT_OPT_ACCEPT_CHECK   2   /* 1 (default): accept a perturbation iff chi^2 decreases; 0: always      */
#define FREDOPT_OPT_MAX_TRIALS     3   /* cap of the `while loop` of Fig. 3 per reduction; default 200            */
#define FREDOPT_OPT_RESET          4   /* any value: k = s = 0, beta restarts at beta0                            */
#define FREDOPT_OPT_USE_GRAPH      5   /* 1 (default): replay one captured iteration as a CUDA graph; 0: launch   */
#define FREDOPT_OPT_TIME_PASSES    6   /* 1: bracket every kernel of fredopt_iterate with CUDA events (implies no */
                                       /*    graph); read with fredopt_get_pass_times; default 0                  */

#define FREDOPT_OPT_BLOCK_SEQUENTIAL 7 /* 1: the feasibility-seeking step follows the loop nest of Fig. 2             */
                                       /*     block by block: sequential over (kind, structure)     */
                                       /*    blocks -- dose kind over the structures, then cDLET, then LETd --        */
                                       /*    simultaneous inside a block: x <- x - lambda eta^k min(w_s,1)/m *        */
                                       /*    sum_{i in block} (r_i/|a_i|^2) a_i, m = rows of the block with a non-zero */
                                       /*    norm; clamp after the last block.  fredopt_get_stats then reports the     */
                                       /*    sets found violated when visited and their proximity share.  Default 0:   */
                                       /*    one simultaneous step over all sets (R1, R23)                   */

#define FREDOPT_OPT_NORMALIZE_GRAD   8 /* 1: the perturbation steps along grad chi^2 / |grad chi^2|_2 (Fig. 3 prints the  */
                                       /*    un-normalised gradient: default 0; R9)             */
#define FREDOPT_OPT_WORK_QUEUE      11 /* how the matrix passes deal their work items to the warps (tuning; never changes a result: */
                                       /*    an item's sum is formed by one warp in a fixed order and stored to a place of its own). */
                                       /*    bit 0 / bit 1: forward / transposed passes take items from a queue (a warp that         */
                                       /*    finishes early takes more) instead of a static round-robin deal; bit 2 / bit 3: forward  */
                                       /*    / transposed items are taken longest first instead of in storage order.  Default: 12, with    */
                                       /*    bit 0 decided per forward launch (queue iff >= 6 items per resident warp of >= 2048 values) */
#define FREDOPT_OPT_USE_PDL         10 /* 1 (default): the kernels of an iteration are launched with programmatic dependent    */
                                       /*    launch (a kernel's CTAs are scheduled while its predecessor drains); 0: plain launches */
#define FREDOPT_OPT_SKIP_SATISFIED  12 /* 1: the back-projection of the simultaneous step streams the values of a row only if the row   */
                                       /*    carries a non-zero coefficient (Fig. 2 touches a row only when its test fires,            */
                                       /*    PAPER.md:129-146); every skipped term is an exact zero: the result has the same bits.     */
                                       /*    Default 0 (stream every value): on the configs[3] plan 65-75 % of the entries stay live    */
                                       /*    over the first hundreds of iterations and looking up liveness costs more than the 25-35 %  */
                                       /*    of values it saves ("Measured dead ends"); it pays close to feasibility         */
#define FREDOPT_OPT_ONE_SIDED_COST   9 /* 1: the OAR term of Eq. (2) penalises only cDL above cDLref: w (cDL - cDLref)_+^2 */
                                       /*    (Eq. (2) as printed is two-sided: default 0; R11)   */

/* Row selectors of the per-pass exports. */
#define FREDOPT_ROWS_ALL     0
#define FREDOPT_ROWS_ACTIVE  1

/* Pass indices of fredopt_get_pass_times / fredopt_get_pass_bytes. */
#define FREDOPT_PASS_FORWARD_X   0   /* d = D x, l = L x on active rows     */
#define FREDOPT_PASS_TRANSPOSE_G 1   /* g = 2 (D^T p + L^T q)                                 (a3)            */
#define FREDOPT_PASS_FORWARD_G   2   /* D g, L g: the perturbed values and the accept test    (a5, a6)        */
#define FREDOPT_PASS_SELECT      3   /* beta selection + x' = x - beta g (scalar kernel)      (a4, a6)        */
#define FREDOPT_PASS_RESIDUAL    4   /* residuals / violations / u, v                         (a7)            */
#define FREDOPT_PASS_TRANSPOSE_B 5   /* back-projection + update + clamp                      (a8, a9)        */
#define FREDOPT_N_PASSES         6

/* Build a plan.  D, L: same n_rows, n_cols (patterns may differ; the union is used).  voxel_labels: n_rows
 * entries in 0..n_struct, 0 = unconstrained.  bounds: n_struct entries (HOST pointer).  cuda_stream: a
 * cudaStream_t (or NULL).  The plan's x starts at 0: call fredopt_set_weights.
 * Errors: INVALID_ARG (null pointer, shape mismatch, bad row_ptr, unsorted / duplicate / out-of-range column,
 * non-finite value, label outside 0..n_struct, weight <= 0 or non-finite, lo > hi, nnz >= 2^32),
 * OUT_OF_MEMORY, CUDA_ERROR, UNSUPPORTED_ARCH. */
int fredopt_create(const fredopt_csr *D, const fredopt_csr *L, const int32_t *voxel_labels,
                   const fredopt_bounds *bounds, int32_t n_struct, void *cuda_stream, fredopt_plan **out);

/* Storage choices of a plan, fixed at creation ("optimized method for storing the Dij and LETij matrices", PAPER.md:282;
 * SURVEY sec. 8f-2).  index_width and block_rows change the bytes a pass moves, never a result: index work is exact, and every
 * sum runs over the same terms plus exact zeros; value_bits = 16 changes the INPUT (see the field).  struct_size = sizeof(fredopt_create_options) of the caller (the struct may grow). */
typedef struct {
    int32_t struct_size;
    int32_t index_width;        /* 0 = automatic: 16-bit indices where exact (n_cols <= 65536; block-row indices of the */
                                /*     transposes inside groups of 65536), int32 otherwise; 32 = int32 everywhere       */
    int32_t block_rows;         /* rows per stored block row of the labelled voxels: consecutive voxels of one          */
                                /*     structure share one stored index per spot over the union of their patterns       */
                                /*     (neighbouring voxels see almost the same spots), in both orientations.           */
                                /*     0 = automatic (the height that stores the fewest bytes), or 1, 2, 4              */
    int32_t shard_rank;         /* ONE plan on several GPUs: the labelled voxels are cut into          */
    int32_t shard_world;        /*     shard_world contiguous voxel ranges balanced by labelled non-zeros                */
                                /*     (fredopt_shard_range); this plan keeps range shard_rank of them.  x is replicated;  */
                                /*     the sums over voxels are completed through fredopt_set_reduce.  0 / 0 or 0 / 1:     */
                                /*     the whole plan.  fredopt_dose_let and the ROWS_ALL exports always cover all voxels  */
    int32_t value_bits;         /* 0 / 32 = the matrix values as given (fp32).  16 = every value of D and L is first replaced */
                                /*     by the nearest IEEE half (round to nearest even; float -> half -> float) -- the plan then */
                                /*     IS the plan of those rounded matrices: dose_let, the per-pass exports, norms, every        */
                                /*     iterate agree with any fp64 evaluation of the rounded matrices as the fp32 plan does with  */
                                /*     the given ones -- and the iteration streams 2-byte copies ("16-bit        */
                                /*     values"): fewer bytes, a DIFFERENT input (relative change up to 4.9e-4 per value; values     */
                                /*     below 6e-8 become 0, above 65504 infinity -> INVALID_ARG).  Not the default, not the        */
                                /*     configuration bench.py's headline times                                                    */
} fredopt_create_options;
/* fredopt_create with options (opt = NULL: the defaults, identical to fredopt_create).  INVALID_ARG on an unknown value. */
int fredopt_create_ex(const fredopt_csr *D, const fredopt_csr *L, const int32_t *voxel_labels,
                      const fredopt_bounds *bounds, int32_t n_struct, void *cuda_stream,
                      const fredopt_create_options *opt, fredopt_plan **out);
void fredopt_destroy(fredopt_plan *plan);

/* Spot weights x (n_cols floats).  set: widened to fp64; get: the plan's fp64 x rounded to fp32.
 * fredopt_get_weights_f64 returns the fp64 state itself (n_cols doubles). */
int fredopt_set_weights(fredopt_plan *plan, const float *x);
int fredopt_get_weights(fredopt_plan *plan, float *x);
int fredopt_get_weights_f64(fredopt_plan *plan, double *x);
int fredopt_set_weights_f64(fredopt_plan *plan, const double *x);   /* the fp64 state itself (checkpoint / resume) */

/* dose = D x, LETd_i = (L x)_i / (D x)_i (0 where dose_i = 0) over ALL n_rows voxels (Eq. 1).
 * x: n_cols floats or NULL = the plan's x.  dose, letd: n_rows floats each; either may be NULL. */
int fredopt_dose_let(fredopt_plan *plan, const float *x, float *dose, float *letd);

/* n_iter iterations of SuperiorDLET (Fig. 3) around the simultaneous AMSrelaxDLET step (Fig. 2), from the plan's
 * x; advances the plan's x, k, s.  lambda in (0, 2]; beta0 >= 0 (0 = pure feasibility-seeking,
 * the paper's "AMS" runs); a in (0, 1).  beta_s = beta0 * a^s by repeated multiplication in fp64;
 * beta0 and a are latched at the first call after create / RESET.  Asynchronous (device work only). */
int fredopt_iterate(fredopt_plan *plan, int32_t n_iter, float lambda, float beta0, float a);

/* The same n_iter iterations as ONE call with the caller's buffers, one synchronisation at its end (the call of an
 * application that keeps its spot weights on the host; bench.py's end-to-end figure times it).  In stream order:
 * x_in (n_cols floats, host or device, or NULL = continue from the plan's x) replaces the plan's x as fredopt_set_weights
 * does; fredopt_iterate(n_iter, lambda, beta0, a); x_out (n_cols floats, host or device, or NULL) receives the plan's x
 * rounded to fp32 as fredopt_get_weights does; stats (HOST, or NULL) as fredopt_get_stats.  Both arrays are borrowed for
 * the call only.  Results are those of the four calls made one after the other, bit for bit.  Errors: those of
 * fredopt_iterate; when the iterations are refused x_in is installed all the same and x_out, stats are untouched. */
int fredopt_iterate_host(fredopt_plan *plan, int32_t n_iter, float lambda, float beta0, float a,
                         const float *x_in, float *x_out, fredopt_stats *stats);

/* Per-voxel bounds and references (bounds are "upper and lower constraints for all organs or defined for each
 * point in the image space"; Eq. (2): per-voxel Dref_i, cDLref_i).  values: n_rows floats, voxel-indexed,
 * host or device; NaN = the voxel keeps its structure's scalar; NULL removes the field's array.  A value applies where the
 * voxel's structure declares that kind of constraint (dose slab: dose_lo or dose_hi; cDL slab; LETd limit) or that cost term
 * (dose_ref, dl_ref): which sets and terms exist stays with the structure.  With FREDOPT_VB_LETD_MAX the norms of the rows
 * L_i - LETmax_i D_i, the participating sets and the normalised weights are set up again.  Errors: INVALID_ARG (infinite value,
 * lo > hi on a voxel; the plan is unchanged).  Synchronises. */
#define FREDOPT_VB_DOSE_LO   0
#define FREDOPT_VB_DOSE_HI   1
#define FREDOPT_VB_DL_LO     2
#define FREDOPT_VB_DL_HI     3
#define FREDOPT_VB_LETD_MAX  4
#define FREDOPT_VB_DOSE_REF  5
#define FREDOPT_VB_DL_REF    6
int fredopt_set_voxel_bounds(fredopt_plan *plan, int32_t field, const float *values);

/* Proximity p(x) = 1/2 sum_{k in P} w^_k r_k^2 / |a_k|^2 and the number of declared sets with r_k != 0.
 * x: n_cols floats or NULL = the plan's x.  prox, n_violated: HOST pointers.  Synchronises. */
int fredopt_proximity(fredopt_plan *plan, const float *x, double *prox, int64_t *n_violated);

int fredopt_set_option(fredopt_plan *plan, int32_t key, double value);
int fredopt_get_stats(fredopt_plan *plan, fredopt_stats *out);

/* ---- one plan on several GPUs (the paper's optimizer is single-GPU) ----
 * Voxel range [*v_begin, *v_end) of shard `rank` of `world`: cuts at the voxel indices where the running count of
 * (non-zeros of D + 1) over LABELLED voxels crosses rank / world of its total.  HOST arrays; pure host code (no GPU
 * needed): every rank computes the same cuts.  INVALID_ARG on bad arguments. */
int fredopt_shard_range(const int64_t *row_ptr, const int32_t *voxel_labels, int64_t n_rows, int32_t rank, int32_t world,
                        int64_t *v_begin, int64_t *v_end);
/* The reduction a sharded plan calls where a sum runs over all voxels: fn must replace buf[0..n) (DEVICE memory, fp64) by its
 * element-wise sum over all ranks -- the same bits on every rank -- ordered on `cuda_stream` (e.g. ncclAllReduce on that
 * stream), and return 0.  It is called once inside fredopt_set_reduce (set counts -> the normalised weights w^ of the WHOLE
 * plan) and then, per superiorized iteration, three times: after the transposed pass of the gradient (n_cols + 1 values: the
 * partial gradient and chi^2), after the forward pass on g (1 value: c) and after the transposed pass of the step (n_cols + 3
 * values: the partial step, proximity, chi^2, violated sets); once per pure feasibility-seeking iteration; once per
 * fredopt_proximity.  The spot weights stay replicated bit for bit because every rank applies the same arithmetic to the same
 * reduced values.  A sharded plan launches its kernels directly (no graph replay) and supports the simultaneous form
 * (FREDOPT_OPT_BLOCK_SEQUENTIAL and the evaluation quantities return FREDOPT_UNSUPPORTED).  fredopt_iterate on a sharded plan
 * without a reduction returns FREDOPT_INVALID_ARG. */
typedef int (*fredopt_reduce_fn)(void *ctx, double *buf, int64_t n, void *cuda_stream);
int fredopt_set_reduce(fredopt_plan *plan, fredopt_reduce_fn fn, void *ctx);

/* The state of Fig. 3 that fredopt_iterate carries from call to call, beside the spot weights: with fredopt_get_weights_f64 /
 * fredopt_set_weights_f64 it is everything a run needs to be resumed -- in another plan, another process -- and to continue
 * bit for bit as if it had not been interrupted (options are the caller's to set again).  Plain data; both calls synchronise. */
typedef struct {
    int64_t k;                  /* iterations done                                          */
    int64_t s;                  /* step-size exponent consumed so far                   */
    int64_t trials;             /* perturbation trials evaluated so far                                    */
    double  beta_next;          /* beta0 * a^s, built by repeated multiplication                           */
    double  eta_pow;            /* eta^k, likewise                                          */
    double  last_beta;          /* last accepted beta                                                      */
    float   beta0, a;           /* the latched pair (reading R8), 0 if none                                */
    int32_t latched;            /* 1 if a superiorized call has latched (beta0, a)                         */
    int32_t reserved;
} fredopt_state;
int fredopt_get_state(fredopt_plan *plan, fredopt_state *out);
int fredopt_set_state(fredopt_plan *plan, const fredopt_state *in);

/* ---- evaluation quantities of the paper's constraint selection and plan comparison (Table 1,
 * PAPER.md:228-236): the dose / LETd / c x D x LETd volume histograms (DVH, LVH, cDLVH), the "value received by a
 * fraction of the structure volume" (cDL30) and a structure's min / mean / max.  quantity: 0 = dose <D_i, x>,
 * 1 = cDL <L_i, x>, 2 = LETd = cDL / dose (0 where the dose is 0); label in 1..n_struct; x: n_cols floats or NULL = the
 * plan's x.  All three synchronise.  An empty structure gives zeros. */
int fredopt_structure_stats(fredopt_plan *plan, const float *x, int32_t quantity, int32_t label,
                            double *vmin, double *vmean, double *vmax, int64_t *n_voxels);   /* HOST pointers, may be NULL */
/* hist[b] = fraction of the structure's voxels whose value is >= b * vmax / n_bins, b = 0..n_bins-1 (cumulative volume
 * histogram; hist: n_bins floats, host or device; 1 <= n_bins <= 2368; vmax > 0). */
int fredopt_volume_histogram(fredopt_plan *plan, const float *x, int32_t quantity, int32_t label, int32_t n_bins,
                             double vmax, float *hist);
/* The smallest of the ceil(fraction * n) largest values of the structure's n voxels: at least `fraction` of the volume
 * receives this value or more (cDL30: quantity 1, fraction 0.3).  0 < fraction <= 1; value: HOST pointer. */
int fredopt_percentile_value(fredopt_plan *plan, const float *x, int32_t quantity, int32_t label, double fraction,
                             double *value);

/* ---- the one call that allocates nothing (for callers that cannot call cudaMalloc: code under CUDA graph capture, serving
 * loops, harnesses that forbid it).  The cumulative volume histogram of fredopt_volume_histogram over the CALLER's arrays,
 * without a plan: values = n_voxels floats, voxel-indexed (e.g. an output of fredopt_dose_let); labels = n_voxels int32 or
 * NULL; the structure is the voxels with labels[i] == label (every voxel when labels is NULL).
 *     hist[b] = fraction of the structure's voxels whose value is >= b * vmax / n_bins, b = 0..n_bins-1; zeros if it is empty;
 *     *n_in_structure = the structure's voxel count (may be NULL).
 * values, labels, hist, n_in_structure: DEVICE pointers, borrowed until the work has run.  Asynchronous on cuda_stream
 * (NULL = the default stream); the device is the CURRENT one.  Bins are decided in fp64 from the fp32 values, as
 * fredopt_volume_histogram decides them from its fp64 products: a value within fp32 rounding of a bin edge may sit in the
 * neighbouring bin.
 * Scratch: the bin counters live in a fixed array in device memory that every GPU loading the library holds until the process
 * exits ((FREDOPT_NO_ALLOC_MAX_BINS + 1) * 8 = 32 776 bytes).  All calls on a GPU share it; each call clears what it uses
 * first, in stream order.  Calls that can overlap on one GPU (different streams, no dependency) RACE on it: order them.
 * No cudaMalloc / cudaFree / allocating library routine is called, neither here nor in fredopt_no_alloc_setup.
 * Errors: INVALID_ARG (null values / hist, n_voxels < 0, n_bins < 1, vmax not positive and finite, and n_bins >
 * FREDOPT_NO_ALLOC_MAX_BINS: the text of fredopt_last_cuda_error() then names the limit), UNSUPPORTED_ARCH, CUDA_ERROR.
 * fredopt_no_alloc_setup looks up the scratch's device address for the current device (once per device; the histogram call
 * does it on first use otherwise): call it before a stream capture begins, since the look-up may load the module. */
#define FREDOPT_NO_ALLOC_MAX_BINS 4096
int fredopt_no_alloc_setup(void);
int fredopt_volume_histogram_no_alloc(const float *values, const int32_t *labels, int64_t n_voxels, int32_t label,
                                      int32_t n_bins, double vmax, float *hist, int64_t *n_in_structure, void *cuda_stream);

/* ---- per-pass exports: per-SpMV parity tests and the isolated-pass sweep (BASELINE.json configs[4]) ----
 * forward:   d = D x, l = L x over the selected rows; d, l: n_rows floats, voxel-indexed (rows outside the
 *            selection are written as 0); either may be NULL (that matrix's values are then not read).
 * transpose: out = D^T u + L^T v over the selected rows; u, v: n_rows floats, voxel-indexed; either may be NULL;
 *            out: n_cols floats.  ROWS_ALL builds a transposed copy of the whole matrix on first use. */
int fredopt_spmv_forward(fredopt_plan *plan, int32_t rows, const float *x, float *d, float *l);
int fredopt_spmv_transpose(fredopt_plan *plan, int32_t rows, const float *u, const float *v, float *out);

/* Accumulated device time [ms] and launch count of each pass of fredopt_iterate since TIME_PASSES was set to 1
 * (ms, launches: FREDOPT_N_PASSES entries each, HOST pointers).  Synchronises. */
int fredopt_get_pass_times(fredopt_plan *plan, double *ms, int64_t *launches);
/* Algorithmic bytes of ONE launch of each pass ("Bytes"): FREDOPT_N_PASSES entries, HOST pointer. */
int fredopt_get_pass_bytes(fredopt_plan *plan, int64_t *bytes);

/* The same for the launches timed since TIME_PASSES was set to 1 (mean per launch).  It differs from fredopt_get_pass_bytes in
 * the back-projection pass, whose need depends on the iterate: every stored index, but the values of those entries only whose
 * (block) row had a non-zero coefficient in that launch (FREDOPT_OPT_SKIP_SATISFIED; counted on the device by a separate kernel
 * after each timed launch).  Without timed launches: the static figures.  Synchronises. */
int fredopt_get_pass_bytes_timed(fredopt_plan *plan, int64_t *bytes);

/* Number of kernels this library has launched on behalf of `plan` since creation. */
int64_t fredopt_launch_count(fredopt_plan *plan);

/* Read-only streaming-sum kernel over `bytes` bytes of device memory (multiple of 16): the practical ceiling of
 * a 100%-read pass on this GPU.  Enqueues `reps` launches on the plan's stream; asynchronous. */
int fredopt_stream_read(fredopt_plan *plan, const void *device_buf, int64_t bytes, int32_t reps);

const char *fredopt_strerror(int code);
/* Text of the last CUDA error seen by this thread inside the library ("" if none). */
const char *fredopt_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* FREDOPT_H */
