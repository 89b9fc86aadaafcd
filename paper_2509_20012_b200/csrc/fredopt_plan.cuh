// fredopt_plan.cuh -- internal declarations shared by the translation units of libfredopt.so:
//   plan_build.cu   fredopt_create: validation, row sets, CSR of the transposes, tables (create time, not hot)
//   iterate.cu      launches of the hot kernels, one iteration of Fig. 3 around Fig. 2, fredopt_iterate, options, state
//   passes.cu       the other calls of include/fredopt.h: weights, dose_let, proximity, per-pass exports, evaluation
// Nothing here touches the CPU oracle; there is no CPU fallback.
#pragma once
#include "../../include/fredopt.h"
#include "fredopt_kernels.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

using namespace fredopt;

// ============================================================================================ errors
extern thread_local std::string g_last_cuda_error;      // defined in passes.cu

#define CK(expr)                                                                                   \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess) {                                                                  \
            g_last_cuda_error = std::string(#expr) + ": " + cudaGetErrorString(e__);               \
            cudaGetLastError();                                                                    \
            return e__ == cudaErrorMemoryAllocation ? FREDOPT_OUT_OF_MEMORY : FREDOPT_CUDA_ERROR;  \
        }                                                                                          \
    } while (0)
#define CKR(expr)                         \
    do {                                  \
        int r__ = (expr);                 \
        if (r__ != FREDOPT_OK) return r__; \
    } while (0)

// ============================================================================================ plan
// A row set in the blocked storage of DESIGN.md "Data layout": n BLOCK ROWS of R consecutive rows each (rows R b + k; the last
// block of a structure may hold fewer than R real rows -- its other rows are padding: vox = -1, rseg = -1).  An ENTRY is one
// (block row, column) pair over the union of the block's column patterns, with R values per matrix (zeros where a row has no
// entry there).  C = 4 / R entries share one 128-bit value load; every block row holds a multiple of C entries (padding:
// column 0, values 0) and starts at a multiple of C; inside every chunk of 32 C entries the entries are interleaved
// (perm_pos in plan_build.cu).
struct RowSet {
    int R = 1;                       // rows per block row (1, 2 or 4)
    long long n = 0;                 // block rows = work items of the forward pass
    long long n_rows = 0;            // n * R: length of every per-row array (d, l, norms, gather vectors, vox, rseg)
    long long n_true = 0;            // real rows
    int n_seg = 1;
    // index / value arrays of the set (block rows stored back to back in list order); exactly one of col / col16 is set
    int32_t* col = nullptr;          // int32 column index per entry
    uint16_t* col16 = nullptr;       // 16-bit form when n_cols <= 65536 (2 B instead of 4 B per entry)
    float* valD = nullptr;           // R values per entry: value k of entry position p at p * R + k
    float* valL = nullptr;
    __half* valD16 = nullptr;        // 16-bit value option: half copies, read by the hot kernels instead of valD / valL
    __half* valL16 = nullptr;
    int32_t* vox = nullptr;          // [n_rows] voxel of the row, -1 = padding
    int16_t* rseg = nullptr;         // [n_rows] structure - 1 of the row, -1 = padding (labelled set only)
    int32_t* seg = nullptr;          // [n] structure - 1 of the block row, or nullptr (one segment)
    long long* start = nullptr;      // [n + 1] first entry position of the block row (multiple of C)
    int32_t* len = nullptr;          // [n] entries, padded to a multiple of C
    int32_t* ulen = nullptr;         // [n] entries of the union pattern
    Item* items = nullptr;           // [n] {start * R, len * R, seg | real rows << 8}: what the forward kernel reads
    Item* items_x = nullptr;         // [n] the same items in execution order (longest first), or nullptr = list order
    int32_t* item_blk = nullptr;     // [n] block row of items_x[e]
    long long nnz = 0;               // non-zeros of the real rows
    long long entries = 0;           // entries of the union patterns (= nnz when R = 1)
    long long entries_padded = 0;
    // CSR of the transposes restricted to this set, SEGMENT-major: run k = (seg * S + spot) * H + group; an entry of a run is
    // one block row (ascending) with its R values per matrix; index = block row (low 16 bits in the 16-bit form)
    bool t_built = false;
    long long* t_ptr = nullptr;      // [n_seg * S * H + 1] entry positions
    int32_t* t_col = nullptr;        // block-row index (32-bit form: only if the 16-bit form does not apply)
    uint16_t* t_col16 = nullptr;     // low 16 bits of the block-row index; runs are cut where the high bits change
    int t_H = 1;                     // number of 65536-block-row groups of the list (1 in the 32-bit form)
    float* t_valD = nullptr;
    float* t_valL = nullptr;
    __half* t_valD16 = nullptr;
    __half* t_valL16 = nullptr;
    long long t_entries_padded = 0;
    // work items of the transposed pass: runs cut into pieces of at most 3 072 (large plans) or TR_ITEM_MAX values per matrix
    long long t_n_items = 0;
    Item* t_items = nullptr;         // [t_n_items] longest first
    int32_t* t_item_slot = nullptr;  // [t_n_items] slot of the item's partial sum
    Item* t_items_run = nullptr;     // [t_n_items] the same items in run (= storage) order
    int32_t* t_slot_run = nullptr;
    long long* t_item_ptr = nullptr; // [S+1] partial-sum slots of spot j: t_item_ptr[j] .. t_item_ptr[j+1]-1
    double* t_partial = nullptr;     // [t_n_items]
    // block-sequential AMS: the same items grouped by structure (longest first inside a structure) and the slot
    // ranges per (spot, structure, group)
    Item* t_items_seg = nullptr;     // [t_n_items]
    int32_t* t_slot_seg = nullptr;   // [t_n_items]
    long long* t_slot_ptr = nullptr; // [S * n_seg * t_H + 1]
    std::vector<long long> t_seg_item_begin;   // host: items of structure s are t_seg_item_begin[s] .. [s+1]-1
    const void* colp() const { return col16 ? (const void*)col16 : (const void*)col; }
};

struct EventPair { cudaEvent_t a, b; int pass; };

struct fredopt_plan {
    cudaStream_t stream = nullptr;
    bool owns_stream = false;
    int device = 0;
    long long V = 0, S = 0, nnz = 0, nnz_padded = 0;
    int n_struct = 0;
    std::vector<void*> allocs;
    // full: all non-empty rows of the padded matrix (union pattern); act: a compact copy of the rows with a label,
    // ordered by (structure, voxel)
    RowSet full, act;
    std::vector<long long> row_base;       // host: rows of structure s are row_base[s] .. row_base[s] + h_tab[s].rows - 1 of `act`
    long long full_class[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};   // rows of length class c of `full`: full_class[c] .. full_class[c+1]-1
    // per active row
    double *nD = nullptr, *nL = nullptr, *nT = nullptr;
    // tables
    StructInfo* tab = nullptr;             // [n_struct]
    std::vector<StructInfo> h_tab;
    uint8_t *mode_union = nullptr, *mode_con = nullptr, *mode_cost = nullptr, *mode_fixed = nullptr;  // mode_fixed: [4][max_seg]
    int max_seg = 1;
    DevState* st = nullptr;
    DevState* st_host = nullptr;           // pinned host copy for fredopt_get_stats (a pageable target would make the copy a staged one)
    VoxBounds vb = {};                     // per-voxel bounds: row-indexed effective values per field (null = structure scalars)
    double* vb_buf[VB_N] = {};             // the arrays behind vb (owned)
    // vectors (fp64)
    double *x = nullptr, *g = nullptr, *xtmp = nullptr;                       // [S]
    float* xstage = nullptr;                                                   // [S] staging of host spot-weight vectors
    double *d = nullptr, *l = nullptr, *Dg = nullptr, *Lg = nullptr;          // [VA]
    GatherVec pq{nullptr, nullptr, nullptr}, uv{nullptr, nullptr, nullptr};    // [VA] gather vectors of the transposed passes
    GatherVec fullUV{nullptr, nullptr, nullptr};                               // lazily: [full.n] gather vector for ROWS_ALL transposes
    double* cpart = nullptr;
    double* gpart = nullptr;                                                   // [ceil(S/256)] partial sums of |g|^2
    double *part_prox = nullptr, *part_phi = nullptr;
    long long* part_cnt = nullptr;
    int* sink = nullptr;
    WorkQueue* wq = nullptr;                                                   // work queue of the item kernels (one launch at a time)
    uint8_t* live8 = nullptr;                                                  // [act.n] 1 iff a row of the block row has a non-zero step coefficient
    unsigned long long* live_count = nullptr;                                  // values the timed back-projections needed (k_count_live)
    int skip_dead = 0;                                                         // back-projection skips block rows without a coefficient (option)
    // options / host state
    double eta = 1.0;
    long long reductionsN = 1, max_trials = 200;
    int accept_check = 1, use_graph = 1, time_passes = 0, block_sequential = 0, normalize_grad = 0, one_sided_cost = 0;
    int use_pdl = 1;
    int fwd_dynamic = -1, tr_dynamic = 0;  // item kernels fed from the work queue (else static round-robin, two waves); -1: per launch
                                           // by item count and length (launch_fwd_kernel)
    int fwd_sorted = 1, tr_sorted = 1;     // items taken longest first (else in storage order)
    bool force_idx32 = false;          // create option: int32 indices in both orientations
    int value_bits = 32;               // create option: 16 = matrix values rounded to IEEE half, half copies for the iteration
    int block_rows_opt = 0;            // create option: rows per block row of the labelled set (0 = chosen by stored bytes)
    int shard_rank = 0, shard_world = 1;   // create option: this plan keeps one voxel range of the labelled rows
    long long shard_begin = 0, shard_end = 0;
    fredopt_reduce_fn reduce_fn = nullptr; // sums a device buffer over all ranks (sharded plans)
    void* reduce_ctx = nullptr;
    double* rbuf = nullptr;            // [S + 8] reduction buffer of the step pass; g has the same 8 spare values
    float* out_stage = nullptr;        // lazily: 2 x n_rows floats staging host outputs of dose_let / spmv_forward
    bool started = false;
    float latched_beta0 = 0.f, latched_a = 0.f;
    cudaError_t launch_err = cudaSuccess;   // first error of a kernel launch since the last check (klaunch)
    long long launches = 0;
    // graphs: [0] = AMS iteration, [1] = SA iteration (for the current reductionsN)
    cudaGraphExec_t gexec[8] = {};       // index = 2 * (2 * block_sequential + (superiorized ? 1 : 0)) + (GRAPH_UNROLL iterations ? 1 : 0)
    long long gexec_red[8] = {};
    int gexec_kernels[8] = {};
    // timing
    std::vector<EventPair> events, event_pool;
    double pass_ms[FREDOPT_N_PASSES] = {0};
    long long pass_launches[FREDOPT_N_PASSES] = {0};
    long long pass_bytes[FREDOPT_N_PASSES] = {0};
    long long tr_con_value_bytes = 0;      // the share of pass_bytes[TRANSPOSE_B] that is matrix values (depends on the iterate)
    long long live_all = -1;               // what k_count_live returns with every block row live (lazily)
    long long live_launches = 0;           // timed back-projections counted into *live_count
    bool count_pending = false;            // a timed back-projection waits for its count (launched by ev_end, outside the bracket)
    const Item* count_items = nullptr;
    const uint8_t* count_mode = nullptr;
    int sm_count = 148;
};


// checked build (fredopt_kernels.cuh, FREDOPT_CHECKED): the extents of every live plan's allocations, mirrored on the device
#ifdef FREDOPT_CHECKED
void chk_register(const void* p, size_t bytes);     // plan_build.cu
void chk_unregister(const void* p);
void chk_sync(cudaStream_t stream);                 // upload the table if it changed (not during a capture)
void chk_upload_iterate(const ChkRange* h, int n);  // one per translation unit that instantiates checked kernels
void chk_upload_passes(const ChkRange* h, int n);
void chk_upload_build(const ChkRange* h, int n);
#else
static inline void chk_register(const void*, size_t) {}
static inline void chk_unregister(const void*) {}
static inline void chk_sync(cudaStream_t) {}
#endif

template <class T>
static inline int dmalloc(fredopt_plan* P, T** p, size_t n) {
    *p = nullptr;
    if (n == 0) n = 1;
    CK(cudaMalloc((void**)p, n * sizeof(T)));
    P->allocs.push_back((void*)*p);
    chk_register((const void*)*p, n * sizeof(T));
    return FREDOPT_OK;
}

static inline int gv_alloc(fredopt_plan* P, GatherVec* g, size_t n) {
    CKR(dmalloc(P, &g->pair, n)); CKR(dmalloc(P, &g->cD, n)); CKR(dmalloc(P, &g->cL, n));
    CK(cudaMemsetAsync(g->pair, 0, (n ? n : 1) * 16, P->stream));
    CK(cudaMemsetAsync(g->cD, 0, (n ? n : 1) * 8, P->stream));
    CK(cudaMemsetAsync(g->cL, 0, (n ? n : 1) * 8, P->stream));
    return FREDOPT_OK;
}

static inline bool is_device_ptr(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

static inline int grid_for(long long n, int threads, int cap) {
    long long g = (n + threads - 1) / threads;
    if (g < 1) g = 1;
    if (g > cap) g = cap;
    return (int)g;
}

// length classes of the full row set (plan_build.cu orders the rows by class; passes.cu launches per class)
constexpr int N_LEN_CLASS = 8, FIRST_SHORT_CLASS = 5;

// ============================================================================================ launches
// Launch one kernel of an iteration on the plan's stream.  With programmatic dependent launch (default) the kernel may be
// scheduled while its predecessor drains; it waits (griddepcontrol.wait at its top) before touching any data.
template <typename... KA, typename... A>
static void klaunch(fredopt_plan* P, void (*kern)(KA...), int grid, int block, A... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = 0; cfg.stream = P->stream;
    cudaLaunchAttribute at;
    at.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &at; cfg.numAttrs = P->use_pdl ? 1 : 0;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, kern, KA(args)...);
    if (e != cudaSuccess && P->launch_err == cudaSuccess) P->launch_err = e;
    ++P->launches;
}

// ---- plan_build.cu
int build_transpose(fredopt_plan* P, RowSet& R);                 // CSR of the transposes of a row set (lazily for ROWS_ALL)
// ---- iterate.cu
int fwd_grid(fredopt_plan* P, long long n);                      // grid of the item kernels (one warp per item, round-robin)
void state_init(fredopt_plan* P);                                // device state at creation
extern const ResidArgs NO_RESID;
void launch_fwd_kernel(fredopt_plan* P, int epi, const RowSet& R, long long b0, long long n, const uint8_t* mode, const double* x,
                       double* oD, double* oL, const GatherVec& pq, const StructInfo* tab, double* cpart, float* fD, float* fL,
                       int letd_out, const ResidArgs& ra);
void launch_forward(fredopt_plan* P, const RowSet& R, const uint8_t* mode, const double* x, double* oD, double* oL, int epi,
                    int write_uv = 0);
void launch_tr_kernel(fredopt_plan* P, const RowSet& R, const Item* items, const int32_t* slots, long long n, const uint8_t* mode,
                      const GatherVec& vec, const uint8_t* live = nullptr);
void launch_transpose(fredopt_plan* P, int tepi, const RowSet& R, const uint8_t* mode, const GatherVec& vec, double* g_out,
                      double* x, float* f_out, const uint8_t* live = nullptr);
void launch_finalize(fredopt_plan* P, int n_part);
void fill_stats(fredopt_plan* P, const DevState& h, fredopt_stats* out);   // iterate.cu: the public statistics from a host copy of the state
void launch_sum_to(fredopt_plan* P, double* out, const double* in, const long long* in_ll, int n);   // out[0] = fixed-order sum
void invalidate_graphs(fredopt_plan* P);
int reduce_call(fredopt_plan* P, double* buf, long long n);      // the caller's reduction on the plan's stream (sharded plans)                         // captured launches hold kernel arguments: capture again
// ---- plan_build.cu
int recount_sets(fredopt_plan* P, bool letd_norms);              // norms of the LETd rows (per-voxel limits), set counts, W, w^
