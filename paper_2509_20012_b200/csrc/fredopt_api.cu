// fredopt_api.cu -- C-ABI (include/fredopt.h), create-time plan builder and pass orchestration.
// The hot kernels are in fredopt_kernels.cuh.  Nothing here touches the CPU oracle; there is no CPU fallback.
#include "../../include/fredopt.h"
#include "fredopt_kernels.cuh"

#include <cub/cub.cuh>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

using namespace fredopt;

// ============================================================================================ errors
static thread_local std::string g_last_cuda_error;

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
// view of a row set for the create-time kernels
struct RowList {
    long long n;                 // rows in the list
    const long long* start;      // [n] offset of the row in the set's padded arrays (multiple of 4)
    const int32_t* len;          // [n] padded length (multiple of 4)
    const int32_t* seg;          // [n] segment (structure - 1), or nullptr = segment 0
    const int32_t* vox;          // [n] voxel index of the row
};

struct RowSet {
    long long n = 0;                 // rows
    int n_seg = 1;
    // padded index / value arrays of the set (rows stored back to back in list order)
    int32_t* col = nullptr;          // int32 column indices (kept for transposition; the hot kernels read col16 if set)
    uint16_t* col16 = nullptr;       // the same indices as 16 bits when n_cols <= 65536 (2 B instead of 4 B per non-zero)
    float* valD = nullptr;
    float* valL = nullptr;
    int32_t* vox = nullptr;          // [n]
    int32_t* seg = nullptr;          // [n] or nullptr
    long long* start = nullptr;      // [n]
    int32_t* len = nullptr;          // [n] padded
    int32_t* ulen = nullptr;         // [n] unpadded
    Item* items = nullptr;           // [n] {start, len, seg}: what the forward kernel reads
    long long nnz = 0;               // unpadded entries in the set
    // CSR of the transposes restricted to this set, SEGMENT-major: run k = seg*S + spot; columns = list index
    bool t_built = false;
    long long* t_ptr = nullptr;      // [n_seg*S + 1]
    int32_t* t_col = nullptr;        // compact row index (32-bit form: only if the 16-bit form does not apply)
    uint16_t* t_col16 = nullptr;     // low 16 bits of the compact row index; runs are cut where the high bits change
    int t_H = 1;                     // number of 65536-row blocks of the list (1 in the 32-bit form)
    float* t_valD = nullptr;
    float* t_valL = nullptr;
    long long t_nnz_padded = 0;
    // work items of the transposed pass: runs cut into pieces of at most TR_ITEM_MAX entries
    long long t_n_items = 0;
    Item* t_items = nullptr;         // [t_n_items]
    int32_t* t_item_slot = nullptr;  // [t_n_items] slot of the item's partial sum
    long long* t_item_ptr = nullptr; // [S+1] partial-sum slots of spot j: t_item_ptr[j] .. t_item_ptr[j+1]-1
    double* t_partial = nullptr;     // [t_n_items]
    // block-sequential AMS: the same items grouped by structure (longest first inside a structure) and the slot
    // ranges per (spot, structure, 65536-row block)
    Item* t_items_seg = nullptr;     // [t_n_items]
    int32_t* t_slot_seg = nullptr;   // [t_n_items]
    long long* t_slot_ptr = nullptr; // [S * n_seg * t_H + 1]
    std::vector<long long> t_seg_item_begin;   // host: items of structure s are t_seg_item_begin[s] .. [s+1]-1
    RowList view() const { return RowList{n, start, len, seg, vox}; }
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
    long long full_class[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};   // rows of length class c of `full`: full_class[c] .. full_class[c+1]-1
    // per active row
    double *nD = nullptr, *nL = nullptr, *nT = nullptr;
    // tables
    StructInfo* tab = nullptr;             // [n_struct]
    std::vector<StructInfo> h_tab;
    uint8_t *mode_union = nullptr, *mode_con = nullptr, *mode_cost = nullptr, *mode_fixed = nullptr;  // mode_fixed: [4][max_seg]
    int max_seg = 1;
    DevState* st = nullptr;
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
    // options / host state
    double eta = 1.0;
    long long reductionsN = 1, max_trials = 200;
    int accept_check = 1, use_graph = 1, time_passes = 0, block_sequential = 0, normalize_grad = 0, one_sided_cost = 0;
    int use_pdl = 1;
    bool started = false;
    float latched_beta0 = 0.f;
    long long launches = 0;
    // graphs: [0] = AMS iteration, [1] = SA iteration (for the current reductionsN)
    cudaGraphExec_t gexec[8] = {};       // index = 2 * (2 * block_sequential + (superiorized ? 1 : 0)) + (GRAPH_UNROLL iterations ? 1 : 0)
    long long gexec_red[8] = {};
    int gexec_kernels[8] = {};
    // timing
    std::vector<EventPair> events;
    double pass_ms[FREDOPT_N_PASSES] = {0};
    long long pass_launches[FREDOPT_N_PASSES] = {0};
    long long pass_bytes[FREDOPT_N_PASSES] = {0};
    int sm_count = 148;
};

template <class T>
static int dmalloc(fredopt_plan* P, T** p, size_t n) {
    *p = nullptr;
    if (n == 0) n = 1;
    CK(cudaMalloc((void**)p, n * sizeof(T)));
    P->allocs.push_back((void*)*p);
    return FREDOPT_OK;
}

static int gv_alloc(fredopt_plan* P, GatherVec* g, size_t n) {
    CKR(dmalloc(P, &g->pair, n)); CKR(dmalloc(P, &g->cD, n)); CKR(dmalloc(P, &g->cL, n));
    CK(cudaMemsetAsync(g->pair, 0, (n ? n : 1) * 16, P->stream));
    CK(cudaMemsetAsync(g->cD, 0, (n ? n : 1) * 8, P->stream));
    CK(cudaMemsetAsync(g->cL, 0, (n ? n : 1) * 8, P->stream));
    return FREDOPT_OK;
}

static bool is_device_ptr(const void* p) {
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

// ============================================================================================ create-time kernels
namespace {

__global__ void k_check_ptr(const long long* ptr, long long V, long long nnz, int* bad) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i <= V; i += (long long)gridDim.x * blockDim.x) {
        const long long a = ptr[i];
        if (a < 0 || a > nnz) *bad = 1;
        if (i == 0 && a != 0) *bad = 1;
        if (i == V && a != nnz) *bad = 1;
        if (i < V && ptr[i + 1] < a) *bad = 1;
    }
}

// warp per row: columns strictly increasing and in range, values finite
__global__ void k_check_rows(const long long* ptr, const int32_t* col, const float* val, long long V, long long S, int* bad) {
    const int lane = threadIdx.x & 31;
    const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long i = w0; i < V; i += nw) {
        const long long b = ptr[i], e = ptr[i + 1];
        for (long long p = b + lane; p < e; p += 32) {
            const int c = col[p];
            if (c < 0 || c >= S) *bad = 2;
            if (p > b && col[p - 1] >= c) *bad = 2;
            if (!isfinite(val[p])) *bad = 3;
        }
    }
}

__global__ void k_check_labels(const int32_t* lab, long long V, int n_struct, int* bad) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += (long long)gridDim.x * blockDim.x)
        if (lab[i] < 0 || lab[i] > n_struct) *bad = 4;
}

__global__ void k_cmp_i64(const long long* a, const long long* b, long long n, int* diff) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        if (a[i] != b[i]) *diff = 1;
}
__global__ void k_cmp_i32(const int32_t* a, const int32_t* b, long long n, int* diff) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        if (a[i] != b[i]) *diff = 1;
}

// union pattern of two sorted rows: count, then fill (thread per row; rare path)
__global__ void k_union_count(const long long* pD, const int32_t* cD, const long long* pL, const int32_t* cL, long long V,
                              long long* cnt) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += (long long)gridDim.x * blockDim.x) {
        long long p = pD[i], pe = pD[i + 1], q = pL[i], qe = pL[i + 1], n = 0;
        while (p < pe || q < qe) {
            const int a = p < pe ? cD[p] : INT32_MAX, b = q < qe ? cL[q] : INT32_MAX;
            if (a == b) { ++p; ++q; } else if (a < b) ++p; else ++q;
            ++n;
        }
        cnt[i] = n;
    }
}
__global__ void k_union_fill(const long long* pD, const int32_t* cD, const float* vD, const long long* pL, const int32_t* cL,
                             const float* vL, long long V, const long long* pU, int32_t* cU, float* uD, float* uL) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += (long long)gridDim.x * blockDim.x) {
        long long p = pD[i], pe = pD[i + 1], q = pL[i], qe = pL[i + 1], o = pU[i];
        while (p < pe || q < qe) {
            const int a = p < pe ? cD[p] : INT32_MAX, b = q < qe ? cL[q] : INT32_MAX;
            if (a == b) { cU[o] = a; uD[o] = vD[p]; uL[o] = vL[q]; ++p; ++q; }
            else if (a < b) { cU[o] = a; uD[o] = vD[p]; uL[o] = 0.f; ++p; }
            else { cU[o] = b; uD[o] = 0.f; uL[o] = vL[q]; ++q; }
            ++o;
        }
    }
}

// per voxel: unpadded length, padded length (as int64 for the scan), flags
__global__ void k_row_lengths(const long long* ptr, const int32_t* lab, long long V, long long* plen64, int32_t* nonempty,
                              int32_t* active) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += (long long)gridDim.x * blockDim.x) {
        const long long n = ptr[i + 1] - ptr[i];
        plen64[i] = (n + 3) & ~3LL;
        nonempty[i] = n > 0;
        active[i] = lab[i] != 0;
    }
}

// compact the flagged voxels (pos = exclusive scan of flag) into a row list
__global__ void k_compact_rows(const int32_t* flag, const int32_t* pos, const long long* ptr, const long long* pstart,
                               const int32_t* lab, long long V, int32_t* vox, long long* start, int32_t* len, int32_t* ulen,
                               int32_t* key) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += (long long)gridDim.x * blockDim.x) {
        if (!flag[i]) continue;
        const int o = pos[i];
        vox[o] = (int32_t)i;
        if (start) {
            const long long n = ptr[i + 1] - ptr[i];
            start[o] = pstart[i];
            len[o] = (int32_t)((n + 3) & ~3LL);
            ulen[o] = (int32_t)n;
        }
        if (key) key[o] = lab[i];
    }
}

// length class of a row of the full set, longest first: 0..4 = more than 1024 / 512 / 256 / 128 / 64 entries (whole warp
// per row; the classes keep the static round-robin balanced), 5 = 33..64 (16 lanes per row), 6 = 17..32 (8 lanes),
// 7 = at most 16 (4 lanes)
constexpr int N_LEN_CLASS = 8, FIRST_SHORT_CLASS = 5;
__host__ __device__ inline int len_class(long long padded) {
    return padded > 1024 ? 0 : padded > 512 ? 1 : padded > 256 ? 2 : padded > 128 ? 3 : padded > 64 ? 4 : padded > 32 ? 5 : padded > 16 ? 6 : 7;
}
__global__ void k_class_keys(const int32_t* vox, const long long* ptr, long long n, int32_t* key, unsigned long long* hist) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n; a += (long long)gridDim.x * blockDim.x) {
        const long long i = vox[a];
        const int c = len_class((ptr[i + 1] - ptr[i] + 3) & ~3LL);
        key[a] = c;
        atomicAdd(hist + c, 1ULL);
    }
}

// after sorting the active voxels by label: fill the list from the voxel ids
__global__ void k_fill_active(const int32_t* vox, const int32_t* lab_sorted, const long long* ptr, const long long* pstart,
                              long long n, long long* start, int32_t* len, int32_t* ulen, int32_t* seg) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n; a += (long long)gridDim.x * blockDim.x) {
        const long long i = vox[a];
        const long long m = ptr[i + 1] - ptr[i];
        start[a] = pstart[i];
        len[a] = (int32_t)((m + 3) & ~3LL);
        ulen[a] = (int32_t)m;
        if (seg) seg[a] = lab_sorted[a] - 1;
    }
}

// Storage order inside a row (or a transposed run) of padded length Lp: every chunk of n <= 128 entries (n a
// multiple of 4, q = n/4 lanes) is interleaved so that memory position 4t+k of the chunk holds the chunk's logical
// entry t + q*k.  A lane's 128-bit load then yields entries t, t+q, t+2q, t+3q, and the k-th gather instruction of
// the warp covers q CONSECUTIVE entries: few cache lines of the gathered vector per instruction.
__device__ __forceinline__ long long perm_pos(long long e, long long Lp) {
    const long long cb = e & ~127LL;
    const long long rem = Lp - cb;
    const int n = rem < 128 ? (int)rem : 128, q = n >> 2, r = (int)(e - cb);
    return cb + 4 * (r % q) + r / q;
}

// copy the rows into the padded arrays (warp per non-empty row); padding stays {col 0, value 0}
__global__ void k_copy_padded(long long n, const int32_t* vox, const long long* start, const long long* ptr, const int32_t* cU,
                              const float* uD, const float* uL, int32_t* col, float* vD, float* vL) {
    const int lane = threadIdx.x & 31;
    const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long r = w0; r < n; r += nw) {
        const long long i = vox[r], b = ptr[i], e = ptr[i + 1], o = start[r];
        const long long Lp = (e - b + 3) & ~3LL;
        for (long long p = b + lane; p < e; p += 32) {
            const long long m = o + perm_pos(p - b, Lp);
            col[m] = cU[p];
            vD[m] = uD[p];
            vL[m] = uL[p];
        }
    }
}

// squared norms of D_i, L_i and L_i - LETmax D_i in fp64 (warp per active row)
__global__ void k_norms(RowList rl, const int32_t* col, const float* vD, const float* vL, const StructInfo* tab, double* nD,
                        double* nL, double* nT) {
    const int lane = threadIdx.x & 31;
    const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long r = w0; r < rl.n; r += nw) {
        const long long s = rl.start[r];
        const int L = rl.len[r];
        const StructInfo& T = tab[rl.seg[r]];
        const double tm = (T.flags & F_LETD) ? T.letd_max : 0.0;
        double a = 0.0, b = 0.0, c = 0.0;
        for (int p = lane; p < L; p += 32) {
            const double dv = (double)vD[s + p], lv = (double)vL[s + p];
            a = fma(dv, dv, a);
            b = fma(lv, lv, b);
            const double t = lv - tm * dv;
            c = fma(t, t, c);
        }
        a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
        if (lane == 0) { nD[r] = a; nL[r] = b; nT[r] = (T.flags & F_LETD) ? c : 0.0; }
    }
}

// integer bookkeeping per structure (atomics on integers: order-independent result)
__global__ void k_count_sets(long long n, const int32_t* seg, const int32_t* ulen, const double* nD, const double* nL,
                             const double* nT, StructInfo* tab) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n; a += (long long)gridDim.x * blockDim.x) {
        StructInfo& T = tab[seg[a]];
        const int f = T.flags;
        unsigned long long sets = 0, part = 0;
        if (f & F_DOSE_SLAB) { ++sets; part += nD[a] > 0.0; if (nD[a] > 0.0) atomicAdd(&T.part_kind[0], 1ULL); }
        if (f & F_DL_SLAB) { ++sets; part += nL[a] > 0.0; if (nL[a] > 0.0) atomicAdd(&T.part_kind[1], 1ULL); }
        if (f & F_LETD) { ++sets; part += nT[a] > 0.0; if (nT[a] > 0.0) atomicAdd(&T.part_kind[2], 1ULL); }
        atomicAdd(&T.n_sets, sets);
        atomicAdd(&T.part, part);
        atomicAdd(&T.n_zero, sets - part);
        atomicAdd(&T.rows, 1ULL);
        atomicAdd(&T.nnz, (unsigned long long)ulen[a]);
    }
}

// W = sum_s w_s * part_s (s ascending), w^_s = w_s / W; pass modes and transposed-pass coefficients
__global__ void k_finish_tables(StructInfo* tab, int n_struct, DevState* st, uint8_t* mode_union, uint8_t* mode_con,
                                uint8_t* mode_cost, uint8_t* mode_fixed, int max_seg) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    double W = 0.0;
    long long ns = 0, nz = 0;
    for (int s = 0; s < n_struct; ++s) { W += tab[s].w * (double)tab[s].part; ns += tab[s].n_sets; nz += tab[s].n_zero; }
    for (int s = 0; s < n_struct; ++s) {
        StructInfo& T = tab[s];
        T.what = W > 0.0 ? T.w / W : 0.0;
        const int f = T.flags;
        const int cost = ((f & F_DOSE_REF) ? 1 : 0) | ((f & F_DL_REF) ? 2 : 0);
        const int con = ((f & (F_DOSE_SLAB | F_LETD)) ? 1 : 0) | ((f & (F_DL_SLAB | F_LETD)) ? 2 : 0);
        mode_cost[s] = (uint8_t)cost;
        mode_con[s] = (uint8_t)con;
        mode_union[s] = (uint8_t)(cost | con);
    }
    for (int s = 0; s < max_seg; ++s) {
        for (int m = 0; m < 4; ++m) mode_fixed[m * max_seg + s] = (uint8_t)m;
    }
    st->W = W; st->n_sets = ns; st->n_zero = nz;
}

// ---- transposition of a row set
// key of an entry = ((segment * S + spot) * H + block) with block = row index >> 16 (H = 1: no blocks)
__global__ void k_tr_keys(RowList rl, const int32_t* ulen, const long long* off, const int32_t* col, long long S, int H,
                          uint32_t* keys, uint32_t* vals) {
    const int lane = threadIdx.x & 31;
    const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long r = w0; r < rl.n; r += nw) {
        const long long s = rl.start[r], o = off[r];
        const int L = ulen[r];
        const int sg = rl.seg ? rl.seg[r] : 0;
        const int Lp = rl.len[r];
        for (int p = lane; p < L; p += 32) {
            keys[o + p] = ((uint32_t)sg * (uint32_t)S + (uint32_t)col[s + perm_pos(p, Lp)]) * (uint32_t)H + (H > 1 ? (uint32_t)(r >> 16) : 0u);
            vals[o + p] = (uint32_t)(o + p);
        }
    }
}
// ustart[k] = first sorted position with key >= k, k = 0..K
__global__ void k_tr_bounds(const uint32_t* keys, long long E, long long K, long long* ustart, long long* pcount) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k <= K; k += (long long)gridDim.x * blockDim.x) {
        long long lo = 0, hi = E;
        while (lo < hi) { const long long mid = (lo + hi) >> 1; if ((long long)keys[mid] < k) lo = mid + 1; else hi = mid; }
        ustart[k] = lo;
    }
}
__global__ void k_tr_pcount(const long long* ustart, long long K, long long* pcount) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < K; k += (long long)gridDim.x * blockDim.x)
        pcount[k] = (ustart[k + 1] - ustart[k] + 3) & ~3LL;
}
__global__ void k_tr_fill(const uint32_t* keys, const uint32_t* vals, long long E, const long long* ustart, const long long* t_ptr,
                          const long long* off, long long n_rows, const long long* start, const int32_t* len, const float* vD,
                          const float* vL, int32_t* t_col, uint16_t* t_col16, float* tD, float* tL) {
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < E; r += (long long)gridDim.x * blockDim.x) {
        const long long k = keys[r], e = vals[r];
        // row a with off[a] <= e < off[a+1]
        long long lo = 0, hi = n_rows;
        while (lo < hi) { const long long mid = (lo + hi) >> 1; if (off[mid + 1] <= e) lo = mid + 1; else hi = mid; }
        const long long a = lo, p = start[a] + perm_pos(e - off[a], len[a]);
        const long long dst = t_ptr[k] + perm_pos(r - ustart[k], t_ptr[k + 1] - t_ptr[k]);
        if (t_col16) t_col16[dst] = (uint16_t)(a & 0xFFFF); else t_col[dst] = (int32_t)a;
        tD[dst] = vD[p];
        tL[dst] = vL[p];
    }
}
// {start, len, seg} -> the 16-byte item the hot kernels read
__global__ void k_pack_items(long long n, const long long* start, const int32_t* len, const int32_t* seg, Item* items) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        Item it;
        it.start = start[i]; it.len = len[i]; it.seg = seg ? seg[i] : 0;
        items[i] = it;
    }
}
// items per (spot, segment) run: ceil(padded length / TR_ITEM_MAX)
__global__ void k_tr_item_count(const long long* t_ptr, long long K, long long* cnt) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < K; k += (long long)gridDim.x * blockDim.x)
        cnt[k] = (t_ptr[k + 1] - t_ptr[k] + TR_ITEM_MAX - 1) / TR_ITEM_MAX;
}
// the same counts in spot-major order (the order of a spot's partial-sum slots)
__global__ void k_tr_item_count_sm(const long long* cnt, long long S, int n_seg, int H, long long* cnt_sm) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < S * n_seg * H; k += (long long)gridDim.x * blockDim.x) {
        const long long hi = k % H, js = k / H, j = js % S, sg = js / S;
        cnt_sm[(j * n_seg + sg) * H + hi] = cnt[k];
    }
}
// item.seg = segment | (block << 8): the kernel adds block << 16 to the 16-bit row indices
__global__ void k_tr_item_fill(const long long* t_ptr, const long long* ibase, const long long* sbase, long long S, int n_seg, int H,
                               Item* items, int32_t* item_slot) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < S * n_seg * H; k += (long long)gridDim.x * blockDim.x) {
        const long long b = t_ptr[k], e = t_ptr[k + 1];
        const long long hi = k % H, js = k / H, j = js % S, sg0 = js / S;
        const long long sg = sg0 | (hi << 8);
        long long i = ibase[k], slot = sbase[(j * n_seg + sg0) * H + hi];
        for (long long p = b; p < e; p += TR_ITEM_MAX, ++i, ++slot) {
            Item it;
            it.start = p; it.len = (int32_t)((e - p) < TR_ITEM_MAX ? (e - p) : TR_ITEM_MAX); it.seg = (int32_t)sg;
            items[i] = it;
            item_slot[i] = (int32_t)slot;
        }
    }
}
// longest-first execution order: key = length class (256-entry bins, longest = 0); a stable sort keeps the
// (structure, spot) order inside a class
__global__ void k_tr_item_key(const Item* items, long long n, uint32_t* key, uint32_t* idx) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        key[i] = (uint32_t)((TR_ITEM_MAX - items[i].len) / 256);
        idx[i] = (uint32_t)i;
    }
}
__global__ void k_tr_item_key_seg(const Item* items, long long n, uint32_t* key, uint32_t* idx, unsigned long long* hist) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const uint32_t sg = (uint32_t)(items[i].seg & 0xFF);
        key[i] = sg * 16u + (uint32_t)((TR_ITEM_MAX - items[i].len) / 256);
        idx[i] = (uint32_t)i;
        atomicAdd(hist + sg, 1ULL);
    }
}
__global__ void k_tr_item_permute(const uint32_t* idx, long long n, const Item* items, const int32_t* js, Item* items2, int32_t* js2) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        items2[i] = items[idx[i]];
        js2[i] = js[idx[i]];
    }
}
__global__ void k_tr_item_ptr(const long long* sbase, long long S, long long runs_per_spot, long long* item_ptr) {
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j <= S; j += (long long)gridDim.x * blockDim.x)
        item_ptr[j] = sbase[j * runs_per_spot];
}
__global__ void k_narrow_u16(const int32_t* in, uint16_t* out, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        out[i] = (uint16_t)in[i];
}
__global__ void k_i32_to_i64(const int32_t* in, long long* out, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) out[i] = in[i];
}

}  // namespace

// ============================================================================================ helpers
template <class T>
static int scan_exclusive(fredopt_plan* P, const T* in, T* out, long long n) {
    size_t tb = 0;
    CK(cub::DeviceScan::ExclusiveSum(nullptr, tb, in, out, n, P->stream));
    void* tmp = nullptr;
    CK(cudaMalloc(&tmp, tb ? tb : 1));
    cudaError_t e = cub::DeviceScan::ExclusiveSum(tmp, tb, in, out, n, P->stream);
    cudaError_t e2 = cudaStreamSynchronize(P->stream);
    cudaFree(tmp);
    CK(e);
    CK(e2);
    return FREDOPT_OK;
}

static int build_transpose(fredopt_plan* P, RowSet& R) {
    cudaStream_t st = P->stream;
    const long long n = R.n, S = P->S;
    // 16-bit row indices: cut every (segment, spot) run where the row index crosses a multiple of 65536
    int H = (int)((n + 65535) >> 16);
    if (H < 1) H = 1;
    bool idx16 = R.n_seg < 256 && H < (1 << 23) && (double)S * R.n_seg * H < 4.0e9 && !getenv("FREDOPT_IDX32");
    if (!idx16) H = 1;
    R.t_H = H;
    const long long K = S * R.n_seg * H;
    // unpadded offsets
    long long *len64 = nullptr, *off = nullptr;
    CK(cudaMalloc(&len64, (n + 1) * sizeof(long long)));
    CK(cudaMalloc(&off, (n + 2) * sizeof(long long)));
    CK(cudaMemsetAsync(len64, 0, (n + 1) * sizeof(long long), st));
    if (n) k_i32_to_i64<<<grid_for(n, 256, 4096), 256, 0, st>>>(R.ulen, len64, n);
    int rc = scan_exclusive(P, len64, off, n + 1);
    cudaFree(len64);
    if (rc) { cudaFree(off); return rc; }
    long long E = 0;
    CK(cudaMemcpyAsync(&E, off + n, sizeof(long long), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    R.nnz = E;
    if (E >= (1LL << 32) || K >= (1LL << 32)) { cudaFree(off); return FREDOPT_INVALID_ARG; }
    uint32_t *keys = nullptr, *vals = nullptr, *keys2 = nullptr, *vals2 = nullptr;
    long long *ustart = nullptr, *pcount = nullptr;
    void* tmp = nullptr;
    int ret = FREDOPT_OK;
    auto cleanup = [&]() {
        cudaFree(keys); cudaFree(vals); cudaFree(keys2); cudaFree(vals2); cudaFree(ustart); cudaFree(pcount); cudaFree(tmp); cudaFree(off);
    };
#define CKC(expr)                                                                                   \
    do {                                                                                            \
        cudaError_t e__ = (expr);                                                                   \
        if (e__ != cudaSuccess) {                                                                   \
            g_last_cuda_error = std::string(#expr) + ": " + cudaGetErrorString(e__);                \
            cudaGetLastError();                                                                     \
            cleanup();                                                                              \
            return e__ == cudaErrorMemoryAllocation ? FREDOPT_OUT_OF_MEMORY : FREDOPT_CUDA_ERROR;   \
        }                                                                                           \
    } while (0)
    const size_t En = E ? (size_t)E : 1;
    CKC(cudaMalloc(&keys, En * 4)); CKC(cudaMalloc(&vals, En * 4));
    CKC(cudaMalloc(&keys2, En * 4)); CKC(cudaMalloc(&vals2, En * 4));
    CKC(cudaMalloc(&ustart, (K + 2) * sizeof(long long))); CKC(cudaMalloc(&pcount, (K + 2) * sizeof(long long)));
    if (n) k_tr_keys<<<grid_for(n * 32, 256, 1 << 16), 256, 0, st>>>(R.view(), R.ulen, off, R.col, S, H, keys, vals);
    int bits = 1;
    while ((1LL << bits) < K) ++bits;
    size_t tb = 0;
    CKC(cub::DeviceRadixSort::SortPairs(nullptr, tb, keys, keys2, vals, vals2, E, 0, bits, st));
    CKC(cudaMalloc(&tmp, tb ? tb : 1));
    CKC(cub::DeviceRadixSort::SortPairs(tmp, tb, keys, keys2, vals, vals2, E, 0, bits, st));   // stable: list order kept inside a key
    k_tr_bounds<<<grid_for(K + 1, 256, 4096), 256, 0, st>>>(keys2, E, K, ustart, pcount);
    CKC(cudaMemsetAsync(pcount, 0, (K + 2) * sizeof(long long), st));
    k_tr_pcount<<<grid_for(K, 256, 4096), 256, 0, st>>>(ustart, K, pcount);
    CKC(cudaGetLastError());
    ret = dmalloc(P, &R.t_ptr, (size_t)K + 2);
    if (ret) { cleanup(); return ret; }
    ret = scan_exclusive(P, pcount, R.t_ptr, K + 1);
    if (ret) { cleanup(); return ret; }
    CKC(cudaMemcpyAsync(&R.t_nnz_padded, R.t_ptr + K, sizeof(long long), cudaMemcpyDeviceToHost, st));
    CKC(cudaStreamSynchronize(st));
    const size_t Tn = R.t_nnz_padded ? (size_t)R.t_nnz_padded : 4;
    if ((ret = idx16 ? dmalloc(P, &R.t_col16, Tn) : dmalloc(P, &R.t_col, Tn)) || (ret = dmalloc(P, &R.t_valD, Tn)) ||
        (ret = dmalloc(P, &R.t_valL, Tn))) { cleanup(); return ret; }
    if (idx16) CKC(cudaMemsetAsync(R.t_col16, 0, Tn * 2, st)); else
    CKC(cudaMemsetAsync(R.t_col, 0, Tn * 4, st));
    CKC(cudaMemsetAsync(R.t_valD, 0, Tn * 4, st));
    CKC(cudaMemsetAsync(R.t_valL, 0, Tn * 4, st));
    if (E) k_tr_fill<<<grid_for(E, 256, 1 << 16), 256, 0, st>>>(keys2, vals2, E, ustart, R.t_ptr, off, n, R.start, R.len, R.valD, R.valL,
                                                             R.t_col, R.t_col16, R.t_valD, R.t_valL);
    CKC(cudaGetLastError());
    // ---- work items: every (segment, spot) run cut into pieces of at most TR_ITEM_MAX entries, in run order
    //      (neighbouring items = neighbouring spots of one structure: overlapping voxel footprints share L1 lines)
    CKC(cudaMemsetAsync(pcount, 0, (K + 2) * sizeof(long long), st));
    k_tr_item_count<<<grid_for(K, 256, 4096), 256, 0, st>>>(R.t_ptr, K, pcount);
    long long *cnt_sm = nullptr, *sbase = nullptr;
    CKC(cudaMalloc(&cnt_sm, (K + 2) * sizeof(long long)));
    { cudaError_t e_ = cudaMalloc(&sbase, (K + 2) * sizeof(long long)); if (e_ != cudaSuccess) { cudaFree(cnt_sm); CKC(e_); } }
    auto cleanup2 = [&]() { cudaFree(cnt_sm); cudaFree(sbase); cleanup(); };
    cudaMemsetAsync(cnt_sm, 0, (K + 2) * sizeof(long long), st);
    k_tr_item_count_sm<<<grid_for(K, 256, 4096), 256, 0, st>>>(pcount, S, R.n_seg, H, cnt_sm);
    ret = scan_exclusive(P, pcount, ustart, K + 1);      // ustart now = first item of each run (execution order)
    if (!ret) ret = scan_exclusive(P, cnt_sm, sbase, K + 1);   // first partial-sum slot of each (spot, segment)
    if (ret) { cleanup2(); return ret; }
    if (cudaMemcpyAsync(&R.t_n_items, ustart + K, sizeof(long long), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) { cleanup2(); return FREDOPT_CUDA_ERROR; }
    if ((ret = dmalloc(P, &R.t_items, (size_t)R.t_n_items)) || (ret = dmalloc(P, &R.t_item_slot, (size_t)R.t_n_items)) ||
        (ret = dmalloc(P, &R.t_item_ptr, (size_t)S + 1)) || (ret = dmalloc(P, &R.t_partial, (size_t)R.t_n_items))) { cleanup2(); return ret; }
    k_tr_item_fill<<<grid_for(K, 256, 4096), 256, 0, st>>>(R.t_ptr, ustart, sbase, S, R.n_seg, H, R.t_items, R.t_item_slot);
    k_tr_item_ptr<<<grid_for(S + 1, 256, 4096), 256, 0, st>>>(sbase, S, (long long)R.n_seg * H, R.t_item_ptr);
    if (cudaGetLastError() != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) { cleanup2(); return FREDOPT_CUDA_ERROR; }
    cudaFree(cnt_sm);
    R.t_slot_ptr = sbase;              // kept: slot ranges per (spot, structure, block) for the block-sequential sweep
    P->allocs.push_back((void*)sbase);
    // ---- the same items grouped by structure, longest first inside a structure (block-sequential AMS)
    R.t_seg_item_begin.assign((size_t)R.n_seg + 1, 0);
    if (R.t_n_items > 0) {
        const long long ni = R.t_n_items;
        uint32_t *ik = nullptr, *ik2 = nullptr, *ii = nullptr, *ii2 = nullptr;
        unsigned long long* hist = nullptr; void* stmp = nullptr;
        auto cleanup4 = [&]() { cudaFree(ik); cudaFree(ik2); cudaFree(ii); cudaFree(ii2); cudaFree(hist); cudaFree(stmp); cleanup(); };
#define CK4(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { g_last_cuda_error = std::string(#expr) + ": " + cudaGetErrorString(e__); cudaGetLastError(); cleanup4(); return e__ == cudaErrorMemoryAllocation ? FREDOPT_OUT_OF_MEMORY : FREDOPT_CUDA_ERROR; } } while (0)
        CK4(cudaMalloc(&ik, ni * 4)); CK4(cudaMalloc(&ik2, ni * 4)); CK4(cudaMalloc(&ii, ni * 4)); CK4(cudaMalloc(&ii2, ni * 4));
        CK4(cudaMalloc(&hist, 256 * 8));
        CK4(cudaMemsetAsync(hist, 0, 256 * 8, st));
        if ((ret = dmalloc(P, &R.t_items_seg, (size_t)ni)) || (ret = dmalloc(P, &R.t_slot_seg, (size_t)ni))) { cleanup4(); return ret; }
        k_tr_item_key_seg<<<grid_for(ni, 256, 4096), 256, 0, st>>>(R.t_items, ni, ik, ii, hist);
        size_t sb = 0;
        CK4(cub::DeviceRadixSort::SortPairs(nullptr, sb, ik, ik2, ii, ii2, ni, 0, 12, st));
        CK4(cudaMalloc(&stmp, sb ? sb : 1));
        CK4(cub::DeviceRadixSort::SortPairs(stmp, sb, ik, ik2, ii, ii2, ni, 0, 12, st));
        k_tr_item_permute<<<grid_for(ni, 256, 4096), 256, 0, st>>>(ii2, ni, R.t_items, R.t_item_slot, R.t_items_seg, R.t_slot_seg);
        unsigned long long hh[256];
        CK4(cudaMemcpyAsync(hh, hist, 256 * 8, cudaMemcpyDeviceToHost, st));
        CK4(cudaStreamSynchronize(st));
#undef CK4
        for (int sg = 0; sg < R.n_seg; ++sg) R.t_seg_item_begin[sg + 1] = R.t_seg_item_begin[sg] + (long long)hh[sg];
        cudaFree(ik); cudaFree(ik2); cudaFree(ii); cudaFree(ii2); cudaFree(hist); cudaFree(stmp);
    }
    // ---- longest items first: with the static round-robin mapping every round of the grid then holds items of
    //      one length class, so the warps stay balanced to within one class width per round
    if (R.t_n_items > 1) {
        const long long ni = R.t_n_items;
        uint32_t *ik = nullptr, *ik2 = nullptr, *ii = nullptr, *ii2 = nullptr;
        Item* it2 = nullptr; int32_t* js2 = nullptr; void* stmp = nullptr;
        auto cleanup3 = [&]() { cudaFree(ik); cudaFree(ik2); cudaFree(ii); cudaFree(ii2); cudaFree(it2); cudaFree(js2); cudaFree(stmp); cleanup(); };
#define CK3(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { g_last_cuda_error = std::string(#expr) + ": " + cudaGetErrorString(e__); cudaGetLastError(); cleanup3(); return e__ == cudaErrorMemoryAllocation ? FREDOPT_OUT_OF_MEMORY : FREDOPT_CUDA_ERROR; } } while (0)
        CK3(cudaMalloc(&ik, ni * 4)); CK3(cudaMalloc(&ik2, ni * 4)); CK3(cudaMalloc(&ii, ni * 4)); CK3(cudaMalloc(&ii2, ni * 4));
        CK3(cudaMalloc(&it2, ni * sizeof(Item))); CK3(cudaMalloc(&js2, ni * sizeof(int32_t)));
        k_tr_item_key<<<grid_for(ni, 256, 4096), 256, 0, st>>>(R.t_items, ni, ik, ii);
        size_t sb = 0;
        CK3(cub::DeviceRadixSort::SortPairs(nullptr, sb, ik, ik2, ii, ii2, ni, 0, 4, st));
        CK3(cudaMalloc(&stmp, sb ? sb : 1));
        CK3(cub::DeviceRadixSort::SortPairs(stmp, sb, ik, ik2, ii, ii2, ni, 0, 4, st));
        k_tr_item_permute<<<grid_for(ni, 256, 4096), 256, 0, st>>>(ii2, ni, R.t_items, R.t_item_slot, it2, js2);
        CK3(cudaMemcpyAsync(R.t_items, it2, ni * sizeof(Item), cudaMemcpyDeviceToDevice, st));
        CK3(cudaMemcpyAsync(R.t_item_slot, js2, ni * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
        CK3(cudaStreamSynchronize(st));
#undef CK3
        cudaFree(ik); cudaFree(ik2); cudaFree(ii); cudaFree(ii2); cudaFree(it2); cudaFree(js2); cudaFree(stmp);
    }
    if (getenv("FREDOPT_DEBUG")) {   // shape of the transposed work list (stderr; debugging aid only)
        std::vector<Item> h((size_t)R.t_n_items);
        cudaMemcpy(h.data(), R.t_items, sizeof(Item) * h.size(), cudaMemcpyDeviceToHost);
        long long hist[8] = {0}, ent[8] = {0};
        for (auto& it : h) { int b = it.len <= 32 ? 0 : it.len <= 128 ? 1 : it.len <= 256 ? 2 : it.len <= 512 ? 3 : it.len <= 1024 ? 4 : it.len < 2048 ? 5 : 6; ++hist[b]; ent[b] += it.len; }
        fprintf(stderr, "[fredopt] transposed set: rows %lld spots %lld segs %d entries %lld padded %lld items %lld\n", n, S, R.n_seg, E, R.t_nnz_padded, R.t_n_items);
        const char* nm[7] = {"<=32", "<=128", "<=256", "<=512", "<=1024", "<2048", "=2048"};
        for (int b = 0; b < 7; ++b) fprintf(stderr, "[fredopt]   len %-6s items %8lld entries %10lld\n", nm[b], hist[b], ent[b]);
    }
    CKC(cudaGetLastError());
    CKC(cudaStreamSynchronize(st));
    cleanup();
#undef CKC
    R.t_built = true;
    return FREDOPT_OK;
}

// bytes the method must move in one launch of a pass: per non-zero 4 B index + 4 B per value array
// the row needs; 8 B per row offset; fp64 vectors read / written once.
static void compute_pass_bytes(fredopt_plan* P) {
    long long fwd_union = 0, fwd_con = 0, tr_cost = 0, tr_con = 0, rows_union = 0, rows_con = 0, rows_cost = 0;
    for (int s = 0; s < P->n_struct; ++s) {
        const StructInfo& T = P->h_tab[s];
        const int f = T.flags;
        const int cost = ((f & F_DOSE_REF) ? 1 : 0) | ((f & F_DL_REF) ? 2 : 0);
        const int con = ((f & (F_DOSE_SLAB | F_LETD)) ? 1 : 0) | ((f & (F_DL_SLAB | F_LETD)) ? 2 : 0);
        auto per = [](int m, int ib) { return m ? ib + 4 * ((m & 1) + ((m >> 1) & 1)) : 0; };
        const int ibf = P->act.col16 ? 2 : 4, ibt = P->act.t_col16 ? 2 : 4;     // index bytes as stored
        fwd_union += (long long)T.nnz * per(cost | con, ibf);
        fwd_con += (long long)T.nnz * per(con, ibf);
        tr_cost += (long long)T.nnz * per(cost, ibt);
        tr_con += (long long)T.nnz * per(con, ibt);
        if (cost | con) rows_union += T.rows;
        if (con) rows_con += T.rows;
        if (cost) rows_cost += T.rows;
    }
    const long long S = P->S, VA = P->act.n;
    P->pass_bytes[FREDOPT_PASS_FORWARD_X] = fwd_union + rows_union * (8 + 16) + S * 8;
    P->pass_bytes[FREDOPT_PASS_FORWARD_G] = fwd_union + rows_union * (8 + 16) + S * 8;
    P->pass_bytes[FREDOPT_PASS_TRANSPOSE_G] = tr_cost + S * P->act.n_seg * 8 + rows_cost * 16 + S * 8;
    P->pass_bytes[FREDOPT_PASS_TRANSPOSE_B] = tr_con + S * P->act.n_seg * 8 + rows_con * 16 + S * 16;
    P->pass_bytes[FREDOPT_PASS_SELECT] = S * 24;
    P->pass_bytes[FREDOPT_PASS_RESIDUAL] = VA * (4 + 8 * 9);
    (void)fwd_con;
}

// ============================================================================================ launches
static void ev_begin(fredopt_plan* P, int pass) {
    if (!P->time_passes) return;
    EventPair ep;
    cudaEventCreate(&ep.a); cudaEventCreate(&ep.b);
    ep.pass = pass;
    cudaEventRecord(ep.a, P->stream);
    P->events.push_back(ep);
}
static void ev_end(fredopt_plan* P) {
    if (!P->time_passes) return;
    cudaEventRecord(P->events.back().b, P->stream);
}

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
    cudaLaunchKernelEx(&cfg, kern, KA(args)...);
    ++P->launches;
}

// grid of the item kernels: one warp per item up to FWD_CTAS_PER_SM resident-CTA-fulls per SM (then round-robin)
constexpr int GRAPH_UNROLL = 8;       // iterations captured into the long graph
constexpr int FWD_CTAS_PER_SM = 2 * FWD_MIN_CTAS;   // 2 waves of the CTAs an SM holds (launch bounds of k_forward / k_transpose)
static int fwd_grid(fredopt_plan* P, long long n) {
    const int cap = P->sm_count * FWD_CTAS_PER_SM < MAX_PARTIALS ? P->sm_count * FWD_CTAS_PER_SM : MAX_PARTIALS;
    return grid_for(n, FWD_WARPS, cap);
}

static const ResidArgs NO_RESID{nullptr, nullptr, nullptr, GatherVec{nullptr, nullptr, nullptr}, nullptr, nullptr, nullptr, nullptr};

// epi: EPI_STORE (d, l), EPI_STORE_PQ (d, l and the cost residuals p, q), EPI_CPART (Dg, Lg and partial sums of c),
// EPI_RESID (d, l and the residual / violation epilogue: step coefficients u, v if write_uv, statistics partials)
static void launch_forward(fredopt_plan* P, const RowSet& R, const uint8_t* mode, const double* x, double* oD, double* oL, int epi,
                           int write_uv = 0) {
    if (R.n == 0) {
        if (epi == EPI_CPART) cudaMemsetAsync(P->cpart, 0, sizeof(double) * MAX_PARTIALS, P->stream);
        if (epi == EPI_RESID) {   // nothing to visit: zero statistics (finalize reads one partial)
            cudaMemsetAsync(P->part_prox, 0, 8, P->stream); cudaMemsetAsync(P->part_phi, 0, 8, P->stream); cudaMemsetAsync(P->part_cnt, 0, 8, P->stream);
            if (write_uv) klaunch(P, k_sweep_end, grid_for(P->S, 256, 1 << 30), 256, P->S, P->x, P->st);   // k, eta^k still advance
        }
        return;
    }
    const int g = fwd_grid(P, R.n);
    const GatherVec none{nullptr, nullptr, nullptr};
    ResidArgs ra = NO_RESID;
    if (epi == EPI_RESID) ra = ResidArgs{P->nD, P->nL, P->nT, write_uv ? P->uv : none, P->part_prox, P->part_phi, P->part_cnt, P->st};
#define FWD_LAUNCH(E, I16, COL, PQ, TAB, CP)                                                                                   \
    klaunch(P, k_forward<E, I16>, g, FWD_THREADS, R.n, R.items, R.vox, mode, COL, R.valD, R.valL, x, oD, oL, PQ, TAB, CP, P->st, \
            nullptr, nullptr, 0, ra)
    if (R.col16) {
        if (epi == EPI_CPART) FWD_LAUNCH(EPI_CPART, true, R.col16, none, P->tab, P->cpart);
        else if (epi == EPI_STORE_PQ) FWD_LAUNCH(EPI_STORE_PQ, true, R.col16, P->pq, P->tab, nullptr);
        else if (epi == EPI_RESID) FWD_LAUNCH(EPI_RESID, true, R.col16, none, P->tab, nullptr);
        else FWD_LAUNCH(EPI_STORE, true, R.col16, none, nullptr, nullptr);
    } else {
        if (epi == EPI_CPART) FWD_LAUNCH(EPI_CPART, false, R.col, none, P->tab, P->cpart);
        else if (epi == EPI_STORE_PQ) FWD_LAUNCH(EPI_STORE_PQ, false, R.col, P->pq, P->tab, nullptr);
        else if (epi == EPI_RESID) FWD_LAUNCH(EPI_RESID, false, R.col, none, P->tab, nullptr);
        else FWD_LAUNCH(EPI_STORE, false, R.col, none, nullptr, nullptr);
    }
#undef FWD_LAUNCH
}
static int cpart_count(fredopt_plan* P) { return P->act.n ? fwd_grid(P, P->act.n) : MAX_PARTIALS; }

template <int EPI>
static void launch_transpose(fredopt_plan* P, const RowSet& R, const uint8_t* mode, const GatherVec& vec, double* g_out, double* x,
                             float* f_out) {
    if (R.t_n_items == 0) return;
    if (R.t_col16)
        klaunch(P, k_transpose<true>, fwd_grid(P, R.t_n_items), FWD_THREADS, R.t_n_items, R.t_items, R.t_item_slot, mode, R.t_col16,
                R.t_valD, R.t_valL, vec, R.t_partial);
    else
        klaunch(P, k_transpose<false>, fwd_grid(P, R.t_n_items), FWD_THREADS, R.t_n_items, R.t_items, R.t_item_slot, mode, R.t_col,
                R.t_valD, R.t_valL, vec, R.t_partial);
    klaunch(P, k_combine<EPI>, grid_for(P->S, 256, 1 << 30), 256, P->S, R.t_item_ptr, R.t_partial, g_out, P->gpart, x, P->st, f_out);
}

static int res_grid(fredopt_plan* P) {
    const int cap = P->sm_count * 4 < MAX_PARTIALS ? P->sm_count * 4 : MAX_PARTIALS;
    const long long n = P->act.n > P->S ? P->act.n : P->S;
    return grid_for(n, ROW_THREADS, cap);
}

static void launch_residual(fredopt_plan* P, double* d, double* l, int use_beta, int final, int write_uv) {
    const int g = res_grid(P);
    klaunch(P, k_residual, g, ROW_THREADS, P->act.n, P->act.items, P->tab, P->st, d, l, P->Dg, P->Lg, P->nD, P->nL, P->nT, P->uv, P->pq,
            P->x, P->g, P->S, P->part_prox, P->part_phi, P->part_cnt, use_beta, final, write_uv);
}

// n_part: how many per-CTA partial sums the last residual pass wrote (k_residual: res_grid; forward epilogue: fwd_grid)
static void launch_finalize(fredopt_plan* P, int n_part) {
    klaunch(P, k_finalize_stats, 1, 1024, P->st, P->part_prox, P->part_phi, P->part_cnt, n_part);
}

// Block-sequential AMS sweep (reading R23): Fig. 2's loop nest -- dose kind over the structures, then cDLET, then the LETd
// rows -- one (forward over the block's rows, residual, transposed over the block's items, update) group per block.
static void enqueue_block_sweep(fredopt_plan* P) {
    const RowSet& A = P->act;
    klaunch(P, k_sweep_begin, 1, 1, P->st);
    std::vector<long long> row_begin((size_t)P->n_struct + 1, 0);
    for (int s = 0; s < P->n_struct; ++s) row_begin[s + 1] = row_begin[s] + (long long)P->h_tab[s].rows;
    const int kind_flag[3] = {F_DOSE_SLAB, F_DL_SLAB, F_LETD};
    const int kind_mode[3] = {1, 2, 3};
    const GatherVec none{nullptr, nullptr, nullptr};
    for (int kind = 0; kind < 3; ++kind)
        for (int s = 0; s < P->n_struct; ++s) {
            const StructInfo& T = P->h_tab[s];
            if (!(T.flags & kind_flag[kind])) continue;
            const long long rb = row_begin[s], re = row_begin[s + 1], nr = re - rb;
            if (nr == 0) continue;
            const uint8_t* md = P->mode_fixed + (size_t)kind_mode[kind] * P->max_seg;
            ev_begin(P, FREDOPT_PASS_FORWARD_X);
            {
                const int g = fwd_grid(P, nr);
                if (A.col16) klaunch(P, k_forward<EPI_STORE, true>, g, FWD_THREADS, nr, A.items + rb, A.vox + rb, md, A.col16, A.valD, A.valL, P->x, P->d + rb, P->l + rb, none, nullptr, nullptr, nullptr, nullptr, nullptr, 0, NO_RESID);
                else klaunch(P, k_forward<EPI_STORE, false>, g, FWD_THREADS, nr, A.items + rb, A.vox + rb, md, A.col, A.valD, A.valL, P->x, P->d + rb, P->l + rb, none, nullptr, nullptr, nullptr, nullptr, nullptr, 0, NO_RESID);
            }
            ev_end(P);
            ev_begin(P, FREDOPT_PASS_RESIDUAL);
            const int gr = grid_for(nr, ROW_THREADS, P->sm_count * 4 < MAX_PARTIALS ? P->sm_count * 4 : MAX_PARTIALS);
            klaunch(P, k_block_residual, gr, ROW_THREADS, rb, re, s, kind, P->tab, P->st, P->d, P->l, P->nD, P->nL, P->nT, P->uv, P->part_prox);
            ev_end(P);
            const long long m = (long long)T.part_kind[kind];
            const long long ib = A.t_seg_item_begin.empty() ? 0 : A.t_seg_item_begin[s], ie = A.t_seg_item_begin.empty() ? 0 : A.t_seg_item_begin[s + 1];
            if (m == 0) continue;                      // no row of the block has a non-zero norm: violations counted, no step
            ev_begin(P, FREDOPT_PASS_TRANSPOSE_B);
            if (ie > ib) {
                const int g = fwd_grid(P, ie - ib);
                if (A.t_col16) klaunch(P, k_transpose<true>, g, FWD_THREADS, ie - ib, A.t_items_seg + ib, A.t_slot_seg + ib, md, A.t_col16, A.t_valD, A.t_valL, P->uv, A.t_partial);
                else klaunch(P, k_transpose<false>, g, FWD_THREADS, ie - ib, A.t_items_seg + ib, A.t_slot_seg + ib, md, A.t_col, A.t_valD, A.t_valL, P->uv, A.t_partial);
            }
            const double factor = (T.w < 1.0 ? T.w : 1.0) / (double)m;
            klaunch(P, k_combine_block, grid_for(P->S, 256, 1 << 30), 256, P->S, A.t_slot_ptr, s, A.n_seg, A.t_H, A.t_partial, P->x, P->st, factor,
                    P->part_prox, gr);
            ev_end(P);
        }
    klaunch(P, k_sweep_end, grid_for(P->S, 256, 1 << 30), 256, P->S, P->x, P->st);
}

// one iteration of Fig. 3 around the simultaneous Fig. 2 step; returns the number of kernels enqueued
static int enqueue_iteration(fredopt_plan* P, bool sa) {
    const long long before = P->launches;
    if (sa) {
        ev_begin(P, FREDOPT_PASS_FORWARD_X);
        launch_forward(P, P->act, P->mode_union, P->x, P->d, P->l, EPI_STORE_PQ);                      // a1, a2: d, l, p, q
        ev_end(P);
        for (long long t = 0; t < P->reductionsN; ++t) {
            ev_begin(P, FREDOPT_PASS_TRANSPOSE_G);
            launch_transpose<TEPI_GRAD>(P, P->act, P->mode_cost, P->pq, P->g, nullptr, nullptr);       // a3: g = D^T p + L^T q
            ev_end(P);
            ev_begin(P, FREDOPT_PASS_FORWARD_G);
            launch_forward(P, P->act, P->mode_union, P->g, P->Dg, P->Lg, EPI_CPART);                   // a5: Dg, Lg, c
            ev_end(P);
            ev_begin(P, FREDOPT_PASS_SELECT);
            klaunch(P, k_select, 1, 1024, P->st, P->gpart, P->act.t_n_items ? grid_for(P->S, 256, 1 << 30) : 0, P->cpart, cpart_count(P), P->act.n,
                    P->act.items, P->tab, P->d, P->l, P->Dg, P->Lg);                                     // a4, a6: beta
            ev_end(P);
            ev_begin(P, FREDOPT_PASS_RESIDUAL);
            const int last = t == P->reductionsN - 1 && !P->block_sequential;
            launch_residual(P, P->d, P->l, 1, last, last);                                             // x', d', l'; a7
            ev_end(P);
        }
    } else if (!P->block_sequential) {      // pure feasibility-seeking: the residual / violation work is the forward pass's epilogue
        ev_begin(P, FREDOPT_PASS_FORWARD_X);
        launch_forward(P, P->act, P->mode_con, P->x, P->d, P->l, EPI_RESID, 1);                       // a1 + a7
        ev_end(P);
    }
    if (P->block_sequential) {
        enqueue_block_sweep(P);
        return (int)(P->launches - before);
    }
    ev_begin(P, FREDOPT_PASS_TRANSPOSE_B);
    launch_transpose<TEPI_UPDATE>(P, P->act, P->mode_con, P->uv, nullptr, P->x, nullptr);              // a8, a9
    ev_end(P);
    return (int)(P->launches - before);
}

// ============================================================================================ API
extern "C" {

const char* fredopt_strerror(int code) {
    switch (code) {
        case FREDOPT_OK: return "ok";
        case FREDOPT_INVALID_ARG: return "invalid argument";
        case FREDOPT_OUT_OF_MEMORY: return "out of device memory";
        case FREDOPT_CUDA_ERROR: return "CUDA error";
        case FREDOPT_UNSUPPORTED_ARCH: return "unsupported GPU architecture (needs compute capability 10.x, built for sm_100a)";
        case FREDOPT_UNSUPPORTED: return "unsupported";
        default: return "unknown error";
    }
}
const char* fredopt_last_cuda_error(void) { return g_last_cuda_error.c_str(); }

void fredopt_destroy(fredopt_plan* P) {
    if (!P) return;
    cudaStreamSynchronize(P->stream);
    for (auto& ep : P->events) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
    for (int i = 0; i < 8; ++i) if (P->gexec[i]) cudaGraphExecDestroy(P->gexec[i]);
    for (void* p : P->allocs) cudaFree(p);
    if (P->owns_stream) cudaStreamDestroy(P->stream);
    delete P;
}

static int create_impl(fredopt_plan* P, const fredopt_csr* D, const fredopt_csr* L, const int32_t* labels,
                       const fredopt_bounds* bounds, int32_t n_struct) {
    cudaStream_t st = P->stream;
    const long long V = D->n_rows, S = D->n_cols;
    P->V = V; P->S = S; P->n_struct = n_struct;
    // ---- host-side table of structures
    P->h_tab.resize(n_struct > 0 ? n_struct : 1);
    for (int s = 0; s < n_struct; ++s) {
        const fredopt_bounds& b = bounds[s];
        if (!(b.weight > 0.f) || !std::isfinite(b.weight)) return FREDOPT_INVALID_ARG;
        if (b.dose_lo > b.dose_hi || b.dl_lo > b.dl_hi) return FREDOPT_INVALID_ARG;
        if (std::isinf(b.dose_lo) || std::isinf(b.dose_hi) || std::isinf(b.dl_lo) || std::isinf(b.dl_hi) || std::isinf(b.letd_max) ||
            std::isinf(b.dose_ref) || std::isinf(b.dl_ref))
            return FREDOPT_INVALID_ARG;
        StructInfo T;
        memset(&T, 0, sizeof(T));
        T.w = (double)b.weight;
        T.dose_lo = (double)b.dose_lo; T.dose_hi = (double)b.dose_hi; T.dl_lo = (double)b.dl_lo; T.dl_hi = (double)b.dl_hi;
        T.letd_max = (double)b.letd_max; T.dose_ref = (double)b.dose_ref; T.dl_ref = (double)b.dl_ref;
        T.flags = ((!std::isnan(b.dose_lo) || !std::isnan(b.dose_hi)) ? F_DOSE_SLAB : 0) |
                  ((!std::isnan(b.dl_lo) || !std::isnan(b.dl_hi)) ? F_DL_SLAB : 0) | (!std::isnan(b.letd_max) ? F_LETD : 0) |
                  (!std::isnan(b.dose_ref) ? F_DOSE_REF : 0) | (!std::isnan(b.dl_ref) ? F_DL_REF : 0);
        P->h_tab[s] = T;
    }
    // ---- inputs on the device (borrowed if already there)
    std::vector<void*> tmp;   // temporaries of this call
    auto tfree = [&]() { for (void* p : tmp) cudaFree(p); tmp.clear(); };
    struct Guard { decltype(tfree)& f; ~Guard() { f(); } } guard{tfree};
    auto to_dev = [&](const void* src, size_t bytes, const void** out) -> int {
        if (bytes == 0) { void* p; CK(cudaMalloc(&p, 16)); tmp.push_back(p); *out = p; return FREDOPT_OK; }
        if (is_device_ptr(src)) { *out = src; return FREDOPT_OK; }
        void* p = nullptr;
        CK(cudaMalloc(&p, bytes));
        tmp.push_back(p);
        CK(cudaMemcpyAsync(p, src, bytes, cudaMemcpyHostToDevice, st));
        *out = p;
        return FREDOPT_OK;
    };
    const long long *pD, *pL; const int32_t *cD, *cL, *lab; const float *vD, *vL;
    CKR(to_dev(D->row_ptr, (V + 1) * 8, (const void**)&pD));
    CKR(to_dev(D->col_idx, D->nnz * 4, (const void**)&cD));
    CKR(to_dev(D->values, D->nnz * 4, (const void**)&vD));
    CKR(to_dev(L->row_ptr, (V + 1) * 8, (const void**)&pL));
    CKR(to_dev(L->col_idx, L->nnz * 4, (const void**)&cL));
    CKR(to_dev(L->values, L->nnz * 4, (const void**)&vL));
    CKR(to_dev(labels, V * 4, (const void**)&lab));
    // ---- validate
    int* flag = nullptr;
    CK(cudaMalloc(&flag, 2 * sizeof(int))); tmp.push_back(flag);
    CK(cudaMemsetAsync(flag, 0, 2 * sizeof(int), st));
    k_check_ptr<<<grid_for(V + 1, 256, 4096), 256, 0, st>>>(pD, V, D->nnz, flag);
    k_check_ptr<<<grid_for(V + 1, 256, 4096), 256, 0, st>>>(pL, V, L->nnz, flag);
    k_check_labels<<<grid_for(V, 256, 4096), 256, 0, st>>>(lab, V, n_struct, flag);
    int hflag[2] = {0, 0};
    CK(cudaMemcpyAsync(hflag, flag, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (hflag[0]) return FREDOPT_INVALID_ARG;
    k_check_rows<<<grid_for(V * 32, 256, 1 << 16), 256, 0, st>>>(pD, cD, vD, V, S, flag);
    k_check_rows<<<grid_for(V * 32, 256, 1 << 16), 256, 0, st>>>(pL, cL, vL, V, S, flag);
    // ---- same pattern?
    int same = D->nnz == L->nnz;
    if (same) {
        k_cmp_i64<<<grid_for(V + 1, 256, 4096), 256, 0, st>>>(pD, pL, V + 1, flag + 1);
        k_cmp_i32<<<grid_for(D->nnz, 256, 1 << 16), 256, 0, st>>>(cD, cL, D->nnz, flag + 1);
    }
    CK(cudaMemcpyAsync(hflag, flag, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    if (hflag[0]) return FREDOPT_INVALID_ARG;
    if (hflag[1]) same = 0;
    const long long* pU = pD; const int32_t* cU = cD; const float *uD = vD, *uL = vL;
    long long nnzU = D->nnz;
    if (!same) {   // union pattern (rare path)
        long long *cnt = nullptr, *pu = nullptr;
        CK(cudaMalloc(&cnt, (V + 1) * 8)); tmp.push_back(cnt);
        CK(cudaMalloc(&pu, (V + 2) * 8)); tmp.push_back(pu);
        CK(cudaMemsetAsync(cnt, 0, (V + 1) * 8, st));
        k_union_count<<<grid_for(V, 128, 1 << 16), 128, 0, st>>>(pD, cD, pL, cL, V, cnt);
        CKR(scan_exclusive(P, cnt, pu, V + 1));
        CK(cudaMemcpyAsync(&nnzU, pu + V, 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        int32_t* cu; float *ud, *ul;
        CK(cudaMalloc(&cu, (nnzU ? nnzU : 1) * 4)); tmp.push_back(cu);
        CK(cudaMalloc(&ud, (nnzU ? nnzU : 1) * 4)); tmp.push_back(ud);
        CK(cudaMalloc(&ul, (nnzU ? nnzU : 1) * 4)); tmp.push_back(ul);
        k_union_fill<<<grid_for(V, 128, 1 << 16), 128, 0, st>>>(pD, cD, vD, pL, cL, vL, V, pu, cu, ud, ul);
        pU = pu; cU = cu; uD = ud; uL = ul;
    }
    if (nnzU >= (1LL << 32)) return FREDOPT_INVALID_ARG;
    P->nnz = nnzU;
    // ---- row lengths, non-empty list, active list
    long long *plen64, *pstart; int32_t *f_ne, *f_act, *pos_ne, *pos_act;
    CK(cudaMalloc(&plen64, (V + 1) * 8)); tmp.push_back(plen64);
    CK(cudaMalloc(&pstart, (V + 2) * 8)); tmp.push_back(pstart);
    CK(cudaMalloc(&f_ne, (V + 1) * 4)); tmp.push_back(f_ne);
    CK(cudaMalloc(&f_act, (V + 1) * 4)); tmp.push_back(f_act);
    CK(cudaMalloc(&pos_ne, (V + 2) * 4)); tmp.push_back(pos_ne);
    CK(cudaMalloc(&pos_act, (V + 2) * 4)); tmp.push_back(pos_act);
    CK(cudaMemsetAsync(plen64, 0, (V + 1) * 8, st));
    CK(cudaMemsetAsync(f_ne, 0, (V + 1) * 4, st));
    CK(cudaMemsetAsync(f_act, 0, (V + 1) * 4, st));
    if (V) k_row_lengths<<<grid_for(V, 256, 1 << 16), 256, 0, st>>>(pU, lab, V, plen64, f_ne, f_act);
    CKR(scan_exclusive(P, plen64, pstart, V + 1));
    CKR(scan_exclusive(P, f_ne, pos_ne, V + 1));
    CKR(scan_exclusive(P, f_act, pos_act, V + 1));
    int32_t n_ne = 0, n_act = 0;
    CK(cudaMemcpyAsync(&P->nnz_padded, pstart + V, 8, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(&n_ne, pos_ne + V, 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(&n_act, pos_act + V, 4, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    // ---- full row set: non-empty rows ordered by (length class, voxel) and stored in that order, so that short rows
    //      (entrance channels, few spots per voxel) are handled by sub-warps over contiguous memory
    RowSet& F = P->full;
    F.n = n_ne; F.n_seg = 1; F.nnz = nnzU;
    CKR(dmalloc(P, &F.vox, (size_t)n_ne)); CKR(dmalloc(P, &F.start, (size_t)n_ne + 1));
    CKR(dmalloc(P, &F.len, (size_t)n_ne)); CKR(dmalloc(P, &F.ulen, (size_t)n_ne)); CKR(dmalloc(P, &F.items, (size_t)n_ne));
    const size_t np = P->nnz_padded ? (size_t)P->nnz_padded : 4;
    CKR(dmalloc(P, &F.col, np)); CKR(dmalloc(P, &F.valD, np)); CKR(dmalloc(P, &F.valL, np));
    CK(cudaMemsetAsync(F.col, 0, np * 4, st)); CK(cudaMemsetAsync(F.valD, 0, np * 4, st)); CK(cudaMemsetAsync(F.valL, 0, np * 4, st));
    {
        int32_t *vox0, *key0, *key1;
        long long *flen64, *fstart;
        unsigned long long* hist;
        CK(cudaMalloc(&vox0, ((size_t)n_ne + 1) * 4)); tmp.push_back(vox0);
        CK(cudaMalloc(&key0, ((size_t)n_ne + 1) * 4)); tmp.push_back(key0);
        CK(cudaMalloc(&key1, ((size_t)n_ne + 1) * 4)); tmp.push_back(key1);
        CK(cudaMalloc(&flen64, ((size_t)n_ne + 1) * 8)); tmp.push_back(flen64);
        CK(cudaMalloc(&fstart, ((size_t)n_ne + 1) * 8)); tmp.push_back(fstart);
        CK(cudaMalloc(&hist, N_LEN_CLASS * 8)); tmp.push_back(hist);
        CK(cudaMemsetAsync(hist, 0, N_LEN_CLASS * 8, st));
        if (V) k_compact_rows<<<grid_for(V, 256, 1 << 16), 256, 0, st>>>(f_ne, pos_ne, pU, pstart, lab, V, vox0, nullptr, nullptr, nullptr, nullptr);
        if (n_ne) k_class_keys<<<grid_for(n_ne, 256, 1 << 16), 256, 0, st>>>(vox0, pU, n_ne, key0, hist);
        size_t tb = 0;
        CK(cub::DeviceRadixSort::SortPairs(nullptr, tb, key0, key1, vox0, F.vox, n_ne, 0, 3, st));
        void* t2; CK(cudaMalloc(&t2, tb ? tb : 1)); tmp.push_back(t2);
        CK(cub::DeviceRadixSort::SortPairs(t2, tb, key0, key1, vox0, F.vox, n_ne, 0, 3, st));   // stable: voxel order inside a class
        if (n_ne) k_fill_active<<<grid_for(n_ne, 256, 1 << 16), 256, 0, st>>>(F.vox, nullptr, pU, pstart, n_ne, fstart, F.len, F.ulen, nullptr);
        CK(cudaMemsetAsync(flen64, 0, ((size_t)n_ne + 1) * 8, st));
        if (n_ne) k_i32_to_i64<<<grid_for(n_ne, 256, 4096), 256, 0, st>>>(F.len, flen64, n_ne);
        CKR(scan_exclusive(P, flen64, F.start, (long long)n_ne + 1));
        unsigned long long hh[N_LEN_CLASS];
        CK(cudaMemcpyAsync(hh, hist, N_LEN_CLASS * 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        P->full_class[0] = 0;
        for (int c = 0; c < N_LEN_CLASS; ++c) P->full_class[c + 1] = P->full_class[c] + (long long)hh[c];
        if (n_ne) {
            k_copy_padded<<<grid_for((long long)n_ne * 32, 256, 1 << 16), 256, 0, st>>>(F.n, F.vox, F.start, pU, cU, uD, uL, F.col, F.valD, F.valL);
            k_pack_items<<<grid_for(n_ne, 256, 4096), 256, 0, st>>>(n_ne, F.start, F.len, nullptr, F.items);
        }
        if (S <= 65536 && !getenv("FREDOPT_IDX32")) {   // 16-bit column indices for the hot kernels
            CKR(dmalloc(P, &F.col16, np));
            k_narrow_u16<<<grid_for((long long)np, 256, 1 << 16), 256, 0, st>>>(F.col, F.col16, (long long)np);
        }
    }
    // ---- active row set, ordered by (label, voxel), with its own compact copy of the rows: the iteration then
    //      streams contiguous arrays (no unconstrained rows in between)
    RowSet& A = P->act;
    A.n = n_act; A.n_seg = n_struct > 0 ? n_struct : 1;
    CKR(dmalloc(P, &A.vox, (size_t)n_act)); CKR(dmalloc(P, &A.start, (size_t)n_act + 1)); CKR(dmalloc(P, &A.len, (size_t)n_act));
    CKR(dmalloc(P, &A.ulen, (size_t)n_act)); CKR(dmalloc(P, &A.seg, (size_t)n_act)); CKR(dmalloc(P, &A.items, (size_t)n_act));
    {
        int32_t *vox0, *key0, *key1;
        long long *alen64, *fstart;
        CK(cudaMalloc(&vox0, (n_act + 1) * 4)); tmp.push_back(vox0);
        CK(cudaMalloc(&key0, (n_act + 1) * 4)); tmp.push_back(key0);
        CK(cudaMalloc(&key1, (n_act + 1) * 4)); tmp.push_back(key1);
        CK(cudaMalloc(&alen64, ((size_t)n_act + 1) * 8)); tmp.push_back(alen64);
        CK(cudaMalloc(&fstart, ((size_t)n_act + 1) * 8)); tmp.push_back(fstart);
        if (V) k_compact_rows<<<grid_for(V, 256, 1 << 16), 256, 0, st>>>(f_act, pos_act, pU, pstart, lab, V, vox0, nullptr, nullptr, nullptr, key0);
        int bits = 1;
        while ((1 << bits) <= n_struct) ++bits;
        size_t tb = 0;
        CK(cub::DeviceRadixSort::SortPairs(nullptr, tb, key0, key1, vox0, A.vox, n_act, 0, bits, st));
        void* t2; CK(cudaMalloc(&t2, tb ? tb : 1)); tmp.push_back(t2);
        CK(cub::DeviceRadixSort::SortPairs(t2, tb, key0, key1, vox0, A.vox, n_act, 0, bits, st));
        // fstart = the row's offset in the full arrays (unused afterwards), A.len / A.ulen / A.seg; then A.start by a scan
        if (n_act) k_fill_active<<<grid_for(n_act, 256, 1 << 16), 256, 0, st>>>(A.vox, key1, pU, pstart, n_act, fstart, A.len, A.ulen, A.seg);
        CK(cudaMemsetAsync(alen64, 0, ((size_t)n_act + 1) * 8, st));
        if (n_act) k_i32_to_i64<<<grid_for(n_act, 256, 4096), 256, 0, st>>>(A.len, alen64, n_act);
        CKR(scan_exclusive(P, alen64, A.start, (long long)n_act + 1));
        long long a_padded = 0;
        CK(cudaMemcpyAsync(&a_padded, A.start + n_act, 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        const size_t na = a_padded ? (size_t)a_padded : 4;
        CKR(dmalloc(P, &A.col, na)); CKR(dmalloc(P, &A.valD, na)); CKR(dmalloc(P, &A.valL, na));
        CK(cudaMemsetAsync(A.col, 0, na * 4, st)); CK(cudaMemsetAsync(A.valD, 0, na * 4, st)); CK(cudaMemsetAsync(A.valL, 0, na * 4, st));
        if (n_act) {
            k_copy_padded<<<grid_for((long long)n_act * 32, 256, 1 << 16), 256, 0, st>>>(A.n, A.vox, A.start, pU, cU, uD, uL, A.col, A.valD, A.valL);
            k_pack_items<<<grid_for(n_act, 256, 4096), 256, 0, st>>>(n_act, A.start, A.len, A.seg, A.items);
        }
        if (S <= 65536 && !getenv("FREDOPT_IDX32")) {
            CKR(dmalloc(P, &A.col16, na));
            k_narrow_u16<<<grid_for((long long)na, 256, 1 << 16), 256, 0, st>>>(A.col, A.col16, (long long)na);
        }
    }
    // ---- tables, norms, w^
    const int ns = n_struct > 0 ? n_struct : 1;
    P->max_seg = ns;
    CKR(dmalloc(P, &P->tab, (size_t)ns));
    CK(cudaMemcpyAsync(P->tab, P->h_tab.data(), sizeof(StructInfo) * ns, cudaMemcpyHostToDevice, st));
    CKR(dmalloc(P, &P->nD, (size_t)n_act)); CKR(dmalloc(P, &P->nL, (size_t)n_act)); CKR(dmalloc(P, &P->nT, (size_t)n_act));
    CKR(dmalloc(P, &P->mode_union, (size_t)ns)); CKR(dmalloc(P, &P->mode_con, (size_t)ns)); CKR(dmalloc(P, &P->mode_cost, (size_t)ns));
    CKR(dmalloc(P, &P->mode_fixed, (size_t)ns * 4));
    CKR(dmalloc(P, &P->st, 1));
    CK(cudaMemsetAsync(P->st, 0, sizeof(DevState), st));
    if (n_act) {
        k_norms<<<grid_for((long long)n_act * 32, 256, 1 << 16), 256, 0, st>>>(A.view(), A.col, A.valD, A.valL, P->tab, P->nD, P->nL, P->nT);
        k_count_sets<<<grid_for(n_act, 256, 4096), 256, 0, st>>>(n_act, A.seg, A.ulen, P->nD, P->nL, P->nT, P->tab);
    }
    k_finish_tables<<<1, 1, 0, st>>>(P->tab, n_struct, P->st, P->mode_union, P->mode_con, P->mode_cost, P->mode_fixed, ns);
    k_set_params<<<1, 1, 0, st>>>(P->st, 1.0, 0.0, 0.5, 1.0, 200, 1, 0, 1);
    CK(cudaMemcpyAsync(P->h_tab.data(), P->tab, sizeof(StructInfo) * ns, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    // ---- vectors
    CKR(dmalloc(P, &P->x, (size_t)S)); CKR(dmalloc(P, &P->g, (size_t)S)); CKR(dmalloc(P, &P->xtmp, (size_t)S));
    CKR(dmalloc(P, &P->xstage, (size_t)S));
    CK(cudaMemsetAsync(P->x, 0, (S ? S : 1) * 8, st)); CK(cudaMemsetAsync(P->g, 0, (S ? S : 1) * 8, st));
    double** vecs[] = {&P->d, &P->l, &P->Dg, &P->Lg};
    for (auto pp : vecs) { CKR(dmalloc(P, pp, (size_t)n_act)); CK(cudaMemsetAsync(*pp, 0, (n_act ? n_act : 1) * 8, st)); }
    CKR(gv_alloc(P, &P->pq, (size_t)n_act)); CKR(gv_alloc(P, &P->uv, (size_t)n_act));
    CKR(dmalloc(P, &P->cpart, (size_t)MAX_PARTIALS));
    CKR(dmalloc(P, &P->gpart, (size_t)(S / 256 + 2)));
    CK(cudaMemsetAsync(P->gpart, 0, (size_t)(S / 256 + 2) * 8, st)); CKR(dmalloc(P, &P->part_prox, (size_t)MAX_PARTIALS));
    CKR(dmalloc(P, &P->part_phi, (size_t)MAX_PARTIALS)); CKR(dmalloc(P, &P->part_cnt, (size_t)MAX_PARTIALS));
    CKR(dmalloc(P, &P->sink, 4));
    CK(cudaMemsetAsync(P->cpart, 0, MAX_PARTIALS * 8, st));
    CK(cudaMemsetAsync(P->part_prox, 0, MAX_PARTIALS * 8, st)); CK(cudaMemsetAsync(P->part_phi, 0, MAX_PARTIALS * 8, st));
    CK(cudaMemsetAsync(P->part_cnt, 0, MAX_PARTIALS * 8, st));
    // ---- CSR of the transposes restricted to the active rows
    CKR(build_transpose(P, A));
    compute_pass_bytes(P);
    CK(cudaStreamSynchronize(st));
    return FREDOPT_OK;
}

int fredopt_create(const fredopt_csr* D, const fredopt_csr* L, const int32_t* voxel_labels, const fredopt_bounds* bounds,
                   int32_t n_struct, void* cuda_stream, fredopt_plan** out) {
    if (!out) return FREDOPT_INVALID_ARG;
    *out = nullptr;
    if (!D || !L || n_struct < 0 || (n_struct > 0 && !bounds)) return FREDOPT_INVALID_ARG;
    if (n_struct > 255) return FREDOPT_UNSUPPORTED;          // work items carry the structure in 8 bits
    if (D->n_rows != L->n_rows || D->n_cols != L->n_cols || D->n_rows < 0 || D->n_cols < 0 || D->nnz < 0 || L->nnz < 0)
        return FREDOPT_INVALID_ARG;
    if (D->n_rows >= (1LL << 31) - 1 || D->n_cols >= (1LL << 31) - 1 || D->nnz >= (1LL << 32) || L->nnz >= (1LL << 32))
        return FREDOPT_INVALID_ARG;
    if (!D->row_ptr || !L->row_ptr || (D->n_rows > 0 && !voxel_labels)) return FREDOPT_INVALID_ARG;
    if ((D->nnz > 0 && (!D->col_idx || !D->values)) || (L->nnz > 0 && (!L->col_idx || !L->values))) return FREDOPT_INVALID_ARG;
    int dev = 0;
    CK(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return FREDOPT_UNSUPPORTED_ARCH;
    fredopt_plan* P = new (std::nothrow) fredopt_plan();
    if (!P) return FREDOPT_OUT_OF_MEMORY;
    P->stream = (cudaStream_t)cuda_stream;
    if (!P->stream) {   // the legacy default stream cannot be captured into a graph: own a blocking stream instead
        cudaError_t e = cudaStreamCreateWithFlags(&P->stream, cudaStreamDefault);
        if (e != cudaSuccess) { delete P; CK(e); }
        P->owns_stream = true;
    }
    P->device = dev;
    P->sm_count = prop.multiProcessorCount;
    if (getenv("FREDOPT_NO_PDL")) P->use_pdl = 0;
    int rc = create_impl(P, D, L, voxel_labels, bounds, n_struct);
    if (rc != FREDOPT_OK) { fredopt_destroy(P); return rc; }
    *out = P;
    return FREDOPT_OK;
}

// ---- host/device staging of small vectors
static int stage_in_f32(fredopt_plan* P, const float* src, size_t n, const float** dev, void** to_free) {
    *to_free = nullptr;
    if (is_device_ptr(src)) { *dev = src; return FREDOPT_OK; }
    void* p = nullptr;
    CK(cudaMalloc(&p, (n ? n : 1) * 4));
    cudaError_t e = cudaMemcpyAsync(p, src, n * 4, cudaMemcpyHostToDevice, P->stream);
    if (e != cudaSuccess) { cudaFree(p); CK(e); }
    *dev = (const float*)p; *to_free = p;
    return FREDOPT_OK;
}

// spot-weight vectors (n_cols floats) from the host go through a staging buffer the plan owns (no allocation per call);
// the copy is complete on return (the caller's array is borrowed for the call only)
static int stage_x(fredopt_plan* P, const float* x, const float** dev) {
    if (is_device_ptr(x)) { *dev = x; return FREDOPT_OK; }
    CK(cudaMemcpyAsync(P->xstage, x, (size_t)P->S * 4, cudaMemcpyHostToDevice, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    *dev = P->xstage;
    return FREDOPT_OK;
}

int fredopt_set_weights(fredopt_plan* P, const float* x) {
    if (!P || !x) return FREDOPT_INVALID_ARG;
    const float* dx;
    CKR(stage_x(P, x, &dx));
    k_f32_to_f64<<<grid_for(P->S, 256, 1024), 256, 0, P->stream>>>(dx, P->x, P->S);
    ++P->launches;
    CK(cudaGetLastError());
    return FREDOPT_OK;
}

int fredopt_get_weights_f64(fredopt_plan* P, double* x) {
    if (!P || !x) return FREDOPT_INVALID_ARG;
    const bool dev = is_device_ptr(x);
    CK(cudaMemcpyAsync(x, P->x, P->S * 8, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, P->stream));
    if (!dev) CK(cudaStreamSynchronize(P->stream));
    return FREDOPT_OK;
}

int fredopt_get_weights(fredopt_plan* P, float* x) {
    if (!P || !x) return FREDOPT_INVALID_ARG;
    if (is_device_ptr(x)) {
        k_f64_to_f32<<<grid_for(P->S, 256, 1024), 256, 0, P->stream>>>(P->x, x, P->S);
        ++P->launches;
        CK(cudaGetLastError());
        return FREDOPT_OK;
    }
    float* tmp = (float*)P->xtmp;   // S doubles of scratch hold S floats
    k_f64_to_f32<<<grid_for(P->S, 256, 1024), 256, 0, P->stream>>>(P->x, tmp, P->S);
    ++P->launches;
    CK(cudaMemcpyAsync(x, tmp, P->S * 4, cudaMemcpyDeviceToHost, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    return FREDOPT_OK;
}

// x argument of dose_let / proximity / spmv_forward: NULL = plan's x, else widened into xtmp
static int resolve_x(fredopt_plan* P, const float* x, const double** xd) {
    if (!x) { *xd = P->x; return FREDOPT_OK; }
    const float* dx;
    CKR(stage_x(P, x, &dx));
    k_f32_to_f64<<<grid_for(P->S, 256, 1024), 256, 0, P->stream>>>(dx, P->xtmp, P->S);
    ++P->launches;
    *xd = P->xtmp;
    return FREDOPT_OK;
}

static int forward_f32(fredopt_plan* P, const RowSet& R, int m, const double* xd, float* d, float* l, int letd_out) {
    // d, l: caller outputs (host or device), voxel-indexed, n_rows floats; rows outside R are 0
    float *dd = d, *dl = l;
    void *fr_d = nullptr, *fr_l = nullptr;
    const size_t nb = (size_t)(P->V ? P->V : 1) * 4;
    if (d && !is_device_ptr(d)) { CK(cudaMalloc(&fr_d, nb)); dd = (float*)fr_d; }
    if (l && !is_device_ptr(l)) { cudaError_t e = cudaMalloc(&fr_l, nb); if (e != cudaSuccess) { cudaFree(fr_d); CK(e); } dl = (float*)fr_l; }
    if (dd) cudaMemsetAsync(dd, 0, (size_t)P->V * 4, P->stream);
    if (dl) cudaMemsetAsync(dl, 0, (size_t)P->V * 4, P->stream);
    if (R.n) {
        const uint8_t* md = P->mode_fixed + (size_t)m * P->max_seg;
        const GatherVec none{nullptr, nullptr, nullptr};
        const bool i16 = R.col16 != nullptr;
        const void* colp = i16 ? (const void*)R.col16 : (const void*)R.col;
        long long n_long = R.n;
        if (&R == &P->full) {   // short rows by sub-warps (4 / 8 / 16 lanes per row), long rows by whole warps
            n_long = P->full_class[FIRST_SHORT_CLASS];
            const long long b[4] = {P->full_class[FIRST_SHORT_CLASS], P->full_class[FIRST_SHORT_CLASS + 1], P->full_class[FIRST_SHORT_CLASS + 2],
                                    P->full_class[FIRST_SHORT_CLASS + 3]};
#define SHORT_LAUNCH(G, LO, HI)                                                                                                  \
    if (HI > LO) {                                                                                                               \
        const int gg = fwd_grid(P, ((HI) - (LO) + (32 / G) - 1) / (32 / G));                                                    \
        if (i16) k_forward_short<G, true><<<gg, FWD_THREADS, 0, P->stream>>>((HI) - (LO), R.items + (LO), R.vox + (LO), m, colp, R.valD, R.valL, xd, dd, dl, letd_out); \
        else k_forward_short<G, false><<<gg, FWD_THREADS, 0, P->stream>>>((HI) - (LO), R.items + (LO), R.vox + (LO), m, colp, R.valD, R.valL, xd, dd, dl, letd_out);    \
        ++P->launches;                                                                                                           \
    }
            SHORT_LAUNCH(16, b[0], b[1])
            SHORT_LAUNCH(8, b[1], b[2])
            SHORT_LAUNCH(4, b[2], b[3])
#undef SHORT_LAUNCH
        }
        if (n_long) {
            if (i16) k_forward<EPI_F32VOX, true><<<fwd_grid(P, n_long), FWD_THREADS, 0, P->stream>>>(n_long, R.items, R.vox, md, colp, R.valD, R.valL, xd, nullptr, nullptr, none, nullptr, nullptr, nullptr, dd, dl, letd_out, NO_RESID);
            else k_forward<EPI_F32VOX, false><<<fwd_grid(P, n_long), FWD_THREADS, 0, P->stream>>>(n_long, R.items, R.vox, md, colp, R.valD, R.valL, xd, nullptr, nullptr, none, nullptr, nullptr, nullptr, dd, dl, letd_out, NO_RESID);
            ++P->launches;
        }
    }
    int rc = FREDOPT_OK;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && fr_d) e = cudaMemcpyAsync(d, dd, (size_t)P->V * 4, cudaMemcpyDeviceToHost, P->stream);
    if (e == cudaSuccess && fr_l) e = cudaMemcpyAsync(l, dl, (size_t)P->V * 4, cudaMemcpyDeviceToHost, P->stream);
    if (fr_d || fr_l) { cudaError_t e2 = cudaStreamSynchronize(P->stream); if (e == cudaSuccess) e = e2; }
    cudaFree(fr_d); cudaFree(fr_l);
    if (e != cudaSuccess) { g_last_cuda_error = cudaGetErrorString(e); cudaGetLastError(); rc = FREDOPT_CUDA_ERROR; }
    return rc;
}

int fredopt_dose_let(fredopt_plan* P, const float* x, float* dose, float* letd) {
    if (!P || (!dose && !letd)) return FREDOPT_INVALID_ARG;
    const double* xd;
    CKR(resolve_x(P, x, &xd));
    return forward_f32(P, P->full, letd ? 3 : 1, xd, dose, letd, 1);
}

int fredopt_spmv_forward(fredopt_plan* P, int32_t rows, const float* x, float* d, float* l) {
    if (!P || (!d && !l) || (rows != FREDOPT_ROWS_ALL && rows != FREDOPT_ROWS_ACTIVE)) return FREDOPT_INVALID_ARG;
    const double* xd;
    CKR(resolve_x(P, x, &xd));
    const RowSet& R = rows == FREDOPT_ROWS_ALL ? P->full : P->act;
    return forward_f32(P, R, (d ? 1 : 0) | (l ? 2 : 0), xd, d, l, 0);
}

int fredopt_spmv_transpose(fredopt_plan* P, int32_t rows, const float* u, const float* v, float* out) {
    if (!P || !out || (!u && !v) || (rows != FREDOPT_ROWS_ALL && rows != FREDOPT_ROWS_ACTIVE)) return FREDOPT_INVALID_ARG;
    RowSet& R = rows == FREDOPT_ROWS_ALL ? P->full : P->act;
    GatherVec vec = P->uv;
    if (rows == FREDOPT_ROWS_ALL) {
        if (!R.t_built) CKR(build_transpose(P, R));
        if (!P->fullUV.pair) CKR(gv_alloc(P, &P->fullUV, (size_t)R.n));
        vec = P->fullUV;
    }
    const float *du = nullptr, *dv = nullptr; void *fu = nullptr, *fv = nullptr;
    if (u) CKR(stage_in_f32(P, u, P->V, &du, &fu));
    if (v) { int rc = stage_in_f32(P, v, P->V, &dv, &fv); if (rc) { cudaFree(fu); return rc; } }
    if (R.n) { k_gather_uv<<<grid_for(R.n, 256, 4096), 256, 0, P->stream>>>(du, dv, R.vox, vec, R.n); ++P->launches; }
    float* dout = out; void* fo = nullptr;
    if (!is_device_ptr(out)) { cudaError_t e = cudaMalloc(&fo, (P->S ? P->S : 1) * 4); if (e != cudaSuccess) { cudaFree(fu); cudaFree(fv); CK(e); } dout = (float*)fo; }
    const int m = (u ? 1 : 0) | (v ? 2 : 0);
    cudaMemsetAsync(dout, 0, (size_t)(P->S ? P->S : 1) * 4, P->stream);     // spots without entries are never visited
    launch_transpose<TEPI_F32>(P, R, P->mode_fixed + (size_t)m * P->max_seg, vec, nullptr, nullptr, dout);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && fo) e = cudaMemcpyAsync(out, dout, P->S * 4, cudaMemcpyDeviceToHost, P->stream);
    if (fo || fu || fv) { cudaError_t e2 = cudaStreamSynchronize(P->stream); if (e == cudaSuccess) e = e2; }
    cudaFree(fo); cudaFree(fu); cudaFree(fv);
    CK(e);
    return FREDOPT_OK;
}

int fredopt_proximity(fredopt_plan* P, const float* x, double* prox, int64_t* n_violated) {
    if (!P || (!prox && !n_violated)) return FREDOPT_INVALID_ARG;
    const double* xd;
    CKR(resolve_x(P, x, &xd));
    // scratch: Dg / Lg hold the products so that the iteration's d, l are left alone
    launch_forward(P, P->act, P->mode_con, xd, P->Dg, P->Lg, EPI_RESID, 0);     // a11: one pass, statistics only
    launch_finalize(P, P->act.n ? fwd_grid(P, P->act.n) : 1);
    DevState h;
    CK(cudaMemcpyAsync(&h, P->st, sizeof(DevState), cudaMemcpyDeviceToHost, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    CK(cudaGetLastError());
    if (prox) *prox = h.prox;
    if (n_violated) *n_violated = h.n_viol;
    return FREDOPT_OK;
}

// ---- evaluation quantities: values of one voxel quantity over the rows of structure `label` into uv.cD[rb .. rb+nr)
static int structure_values(fredopt_plan* P, const float* x, int32_t quantity, int32_t label, long long* rb_out, long long* nr_out) {
    if (!P || quantity < 0 || quantity > 2 || label < 1 || label > P->n_struct) return FREDOPT_INVALID_ARG;
    const double* xd;
    CKR(resolve_x(P, x, &xd));
    long long rb = 0;
    for (int s = 0; s < label - 1; ++s) rb += (long long)P->h_tab[s].rows;
    const long long nr = (long long)P->h_tab[label - 1].rows;
    *rb_out = rb; *nr_out = nr;
    if (nr == 0) return FREDOPT_OK;
    const RowSet& A = P->act;
    const int m = quantity == 0 ? 1 : quantity == 1 ? 2 : 3;
    const uint8_t* md = P->mode_fixed + (size_t)m * P->max_seg;
    const GatherVec none{nullptr, nullptr, nullptr};
    const int g = fwd_grid(P, nr);
    if (A.col16) k_forward<EPI_STORE, true><<<g, FWD_THREADS, 0, P->stream>>>(nr, A.items + rb, A.vox + rb, md, A.col16, A.valD, A.valL, xd, P->Dg + rb, P->Lg + rb, none, nullptr, nullptr, nullptr, nullptr, nullptr, 0, NO_RESID);
    else k_forward<EPI_STORE, false><<<g, FWD_THREADS, 0, P->stream>>>(nr, A.items + rb, A.vox + rb, md, A.col, A.valD, A.valL, xd, P->Dg + rb, P->Lg + rb, none, nullptr, nullptr, nullptr, nullptr, nullptr, 0, NO_RESID);
    k_quantity<<<grid_for(nr, 256, 1024), 256, 0, P->stream>>>(nr, quantity, P->Dg + rb, P->Lg + rb, P->uv.cD + rb);
    P->launches += 2;
    CK(cudaGetLastError());
    return FREDOPT_OK;
}

int fredopt_structure_stats(fredopt_plan* P, const float* x, int32_t quantity, int32_t label, double* vmin, double* vmean,
                            double* vmax, int64_t* n_voxels) {
    long long rb, nr;
    CKR(structure_values(P, x, quantity, label, &rb, &nr));
    double h[3] = {0.0, 0.0, 0.0};
    if (nr) {
        k_value_stats<<<1, 1024, 0, P->stream>>>(nr, P->uv.cD + rb, P->part_prox);
        ++P->launches;
        CK(cudaMemcpyAsync(h, P->part_prox, 3 * sizeof(double), cudaMemcpyDeviceToHost, P->stream));
        CK(cudaStreamSynchronize(P->stream));
        h[1] /= (double)nr;
    }
    if (vmin) *vmin = h[0];
    if (vmean) *vmean = h[1];
    if (vmax) *vmax = h[2];
    if (n_voxels) *n_voxels = nr;
    return FREDOPT_OK;
}

int fredopt_volume_histogram(fredopt_plan* P, const float* x, int32_t quantity, int32_t label, int32_t n_bins, double vmax,
                             float* hist) {
    if (!hist || n_bins < 1 || n_bins > MAX_PARTIALS || !(vmax > 0.0) || !std::isfinite(vmax)) return FREDOPT_INVALID_ARG;
    long long rb, nr;
    CKR(structure_values(P, x, quantity, label, &rb, &nr));
    std::vector<unsigned long long> c((size_t)n_bins, 0ULL);
    if (nr) {
        CK(cudaMemsetAsync(P->part_cnt, 0, (size_t)n_bins * 8, P->stream));
        k_value_hist<<<grid_for(nr, 256, 1024), 256, 0, P->stream>>>(nr, P->uv.cD + rb, n_bins, vmax, (unsigned long long*)P->part_cnt);
        ++P->launches;
        CK(cudaMemcpyAsync(c.data(), P->part_cnt, (size_t)n_bins * 8, cudaMemcpyDeviceToHost, P->stream));
        CK(cudaStreamSynchronize(P->stream));
    }
    std::vector<float> hh((size_t)n_bins, 0.f);
    unsigned long long cum = 0;
    for (int b = n_bins - 1; b >= 0; --b) { cum += c[b]; hh[b] = nr ? (float)((double)cum / (double)nr) : 0.f; }
    if (is_device_ptr(hist)) { CK(cudaMemcpyAsync(hist, hh.data(), (size_t)n_bins * 4, cudaMemcpyHostToDevice, P->stream)); CK(cudaStreamSynchronize(P->stream)); }
    else memcpy(hist, hh.data(), (size_t)n_bins * 4);
    return FREDOPT_OK;
}

int fredopt_percentile_value(fredopt_plan* P, const float* x, int32_t quantity, int32_t label, double fraction, double* value) {
    if (!value || !(fraction > 0.0) || !(fraction <= 1.0)) return FREDOPT_INVALID_ARG;
    long long rb, nr;
    CKR(structure_values(P, x, quantity, label, &rb, &nr));
    *value = 0.0;
    if (nr == 0) return FREDOPT_OK;
    size_t tb = 0;
    CK(cub::DeviceRadixSort::SortKeysDescending(nullptr, tb, P->uv.cD + rb, P->uv.cL + rb, nr, 0, 64, P->stream));
    void* tmp = nullptr;
    CK(cudaMalloc(&tmp, tb ? tb : 1));
    cudaError_t e = cub::DeviceRadixSort::SortKeysDescending(tmp, tb, P->uv.cD + rb, P->uv.cL + rb, nr, 0, 64, P->stream);
    long long k = (long long)std::ceil(fraction * (double)nr);
    if (k < 1) k = 1;
    if (k > nr) k = nr;
    if (e == cudaSuccess) e = cudaMemcpyAsync(value, P->uv.cL + rb + (k - 1), sizeof(double), cudaMemcpyDeviceToHost, P->stream);
    cudaError_t e2 = cudaStreamSynchronize(P->stream);
    cudaFree(tmp);
    ++P->launches;
    CK(e); CK(e2);
    return FREDOPT_OK;
}

int fredopt_set_option(fredopt_plan* P, int32_t key, double value) {
    if (!P) return FREDOPT_INVALID_ARG;
    switch (key) {
        case FREDOPT_OPT_ETA: if (!(value > 0.0) || value > 1.0) return FREDOPT_INVALID_ARG; P->eta = value; break;
        case FREDOPT_OPT_REDUCTIONS:
            if (value < 1.0 || value > 1000.0) return FREDOPT_INVALID_ARG;
            P->reductionsN = (long long)value;
            break;
        case FREDOPT_OPT_ACCEPT_CHECK: P->accept_check = value != 0.0; break;
        case FREDOPT_OPT_MAX_TRIALS: if (value < 1.0) return FREDOPT_INVALID_ARG; P->max_trials = (long long)value; break;
        case FREDOPT_OPT_RESET: {
            P->started = false;
            DevState h;
            CK(cudaMemcpyAsync(&h, P->st, sizeof(DevState), cudaMemcpyDeviceToHost, P->stream));
            CK(cudaStreamSynchronize(P->stream));
            h.k = 0; h.s = 0; h.trials = 0; h.last_beta = 0.0; h.eta_pow = 1.0; h.beta_acc = 0.0;
            CK(cudaMemcpyAsync(P->st, &h, sizeof(DevState), cudaMemcpyHostToDevice, P->stream));
            CK(cudaStreamSynchronize(P->stream));
            break;
        }
        case FREDOPT_OPT_USE_GRAPH: P->use_graph = value != 0.0; break;
        case FREDOPT_OPT_BLOCK_SEQUENTIAL: P->block_sequential = value != 0.0; break;
        case FREDOPT_OPT_NORMALIZE_GRAD: P->normalize_grad = value != 0.0; break;
        case FREDOPT_OPT_ONE_SIDED_COST: P->one_sided_cost = value != 0.0; break;
        case FREDOPT_OPT_TIME_PASSES:
            P->time_passes = value != 0.0;
            if (P->time_passes) {
                for (auto& ep : P->events) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
                P->events.clear();
                for (int i = 0; i < FREDOPT_N_PASSES; ++i) { P->pass_ms[i] = 0; P->pass_launches[i] = 0; }
            }
            break;
        default: return FREDOPT_INVALID_ARG;
    }
    return FREDOPT_OK;
}

int fredopt_iterate(fredopt_plan* P, int32_t n_iter, float lambda, float beta0, float a) {
    if (!P || n_iter < 0) return FREDOPT_INVALID_ARG;
    if (!(lambda > 0.f) || !(lambda <= 2.f) || !(beta0 >= 0.f) || !std::isfinite(beta0) || !(a > 0.f) || !(a < 1.f))
        return FREDOPT_INVALID_ARG;
    const int latch = !P->started;
    if (latch) { P->latched_beta0 = beta0; P->started = true; }
    k_set_params<<<1, 1, 0, P->stream>>>(P->st, (double)lambda, (double)beta0, (double)a, P->eta, P->max_trials, P->accept_check,
                                           (P->normalize_grad ? SF_NORMALIZE_GRAD : 0) | (P->one_sided_cost ? SF_ONE_SIDED : 0), latch);
    ++P->launches;
    const bool sa = beta0 != 0.f;
    if (n_iter > 0) {
        const bool graph = P->use_graph && !P->time_passes;
        if (graph) {
            // two graphs per form: one iteration, and GRAPH_UNROLL iterations back to back (fewer graph launches for the
            // small plans, whose iteration lasts about as long as a graph launch costs)
            const int form = 2 * P->block_sequential + (sa ? 1 : 0);
            int left = n_iter;
            // (measured: +3 % on configs[0]-[1], +1 % on configs[2], nothing at configs[3]: long graph only below 5e7 non-zeros)
            for (int u = P->act.nnz < 50000000LL ? 1 : 0; u >= 0; --u) {
                const int per = u ? GRAPH_UNROLL : 1, gi = 2 * form + u;
                // both graphs are built at the first call of a form, so that no later (timed) call pays for a capture
                if (!P->gexec[gi] || P->gexec_red[gi] != P->reductionsN) {
                    if (P->gexec[gi]) { cudaGraphExecDestroy(P->gexec[gi]); P->gexec[gi] = nullptr; }
                    cudaGraph_t gr = nullptr;
                    CK(cudaStreamBeginCapture(P->stream, cudaStreamCaptureModeThreadLocal));
                    const long long l0 = P->launches;
                    int nk = 0;
                    for (int r = 0; r < per; ++r) nk += enqueue_iteration(P, sa);
                    P->launches = l0;
                    cudaError_t e = cudaStreamEndCapture(P->stream, &gr);
                    CK(e);
                    e = cudaGraphInstantiate(&P->gexec[gi], gr, 0);
                    cudaGraphDestroy(gr);
                    CK(e);
                    P->gexec_red[gi] = P->reductionsN;
                    P->gexec_kernels[gi] = nk;
                }
                for (; left >= per; left -= per) { CK(cudaGraphLaunch(P->gexec[gi], P->stream)); P->launches += P->gexec_kernels[gi]; }
            }
        } else {
            for (int it = 0; it < n_iter; ++it) enqueue_iteration(P, sa);
        }
        if (!P->block_sequential)                         // block mode keeps its sweep statistics in the state already
            launch_finalize(P, sa ? res_grid(P) : (P->act.n ? fwd_grid(P, P->act.n) : 1));
    }
    CK(cudaGetLastError());
    return FREDOPT_OK;
}

int fredopt_get_stats(fredopt_plan* P, fredopt_stats* out) {
    if (!P || !out) return FREDOPT_INVALID_ARG;
    DevState h;
    CK(cudaMemcpyAsync(&h, P->st, sizeof(DevState), cudaMemcpyDeviceToHost, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    out->k = h.k; out->s = h.s; out->trials = h.trials; out->n_violated = h.n_viol;
    out->n_sets = h.n_sets; out->n_zero_norm_sets = h.n_zero;
    out->n_active_rows = P->act.n; out->nnz = P->nnz; out->nnz_active = P->act.nnz;
    long long b = 0;
    const int sa_passes[] = {FREDOPT_PASS_FORWARD_X, FREDOPT_PASS_TRANSPOSE_G, FREDOPT_PASS_FORWARD_G, FREDOPT_PASS_SELECT,
                             FREDOPT_PASS_RESIDUAL, FREDOPT_PASS_TRANSPOSE_B};
    for (int p : sa_passes) b += P->pass_bytes[p];
    out->alg_bytes_iter = b;
    out->last_beta = h.last_beta; out->phi = h.phi; out->prox = h.prox; out->weight_sum = h.W;
    return FREDOPT_OK;
}

int fredopt_get_pass_times(fredopt_plan* P, double* ms, int64_t* launches) {
    if (!P || !ms || !launches) return FREDOPT_INVALID_ARG;
    CK(cudaStreamSynchronize(P->stream));
    for (auto& ep : P->events) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, ep.a, ep.b) == cudaSuccess) { P->pass_ms[ep.pass] += t; P->pass_launches[ep.pass] += 1; }
        cudaEventDestroy(ep.a); cudaEventDestroy(ep.b);
    }
    cudaGetLastError();
    P->events.clear();
    for (int i = 0; i < FREDOPT_N_PASSES; ++i) { ms[i] = P->pass_ms[i]; launches[i] = P->pass_launches[i]; }
    return FREDOPT_OK;
}

int fredopt_get_pass_bytes(fredopt_plan* P, int64_t* bytes) {
    if (!P || !bytes) return FREDOPT_INVALID_ARG;
    for (int i = 0; i < FREDOPT_N_PASSES; ++i) bytes[i] = P->pass_bytes[i];
    return FREDOPT_OK;
}

int64_t fredopt_launch_count(fredopt_plan* P) { return P ? P->launches : 0; }

int fredopt_stream_read(fredopt_plan* P, const void* device_buf, int64_t bytes, int32_t reps) {
    if (!P || !device_buf || bytes < 16 || (bytes & 15) || reps < 1 || !is_device_ptr(device_buf)) return FREDOPT_INVALID_ARG;
    for (int i = 0; i < reps; ++i) {
        k_stream_read<<<(unsigned)((bytes / 16 + 2047) / 2048), 256, 0, P->stream>>>((const int4*)device_buf, bytes / 16, P->sink);
        ++P->launches;
    }
    CK(cudaGetLastError());
    return FREDOPT_OK;
}

}  // extern "C"
