// plan_build.cu -- fredopt_create: validation of the inputs, the row sets (all non-empty rows; a compact copy of the labelled
// rows), padding + interleave, 16-bit indices, norms, weight normalisation, the stored CSR of the transposes with its work
// items and slots, algorithmic byte counts.  Create time only: nothing here runs inside fredopt_iterate.
#include "fredopt_plan.cuh"

#include <cub/cub.cuh>

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

// 16-bit value storage (fredopt_create_options.value_bits = 16): every stored value is replaced by the nearest IEEE half (round to
// nearest even, the conversion numpy and every IEEE library perform), in place in fp32 -- norms, tables and the fp32 row sets then
// see exactly the values the half copies hold -- and the hot arrays get half copies
__global__ void k_round_to_half(float* v, size_t n, int* overflow) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float r = __half2float(__float2half_rn(v[i]));
        if (isinf(r)) *overflow = 1;                                 // |value| > 65504 (inputs are finite: checked before)
        v[i] = r;
    }
}
__global__ void k_to_half(const float* v, __half* h, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) h[i] = __float2half_rn(v[i]);
}
// per voxel: padded length of the row as a block row of its own (multiple of 4; int64 for the scan), flags
__global__ void k_row_lengths(const long long* ptr, const int32_t* lab, long long V, long long vb, long long ve, int32_t* nonempty,
                              int32_t* active) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += (long long)gridDim.x * blockDim.x) {
        nonempty[i] = ptr[i + 1] > ptr[i];
        active[i] = lab[i] != 0 && i >= vb && i < ve;      // a sharded plan keeps the labelled voxels of its range
    }
}

// compact the flagged voxels (pos = exclusive scan of flag) into a list; key = label (optional)
__global__ void k_compact_rows(const int32_t* flag, const int32_t* pos, const int32_t* lab, long long V, int32_t* vox, int32_t* key) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < V; i += (long long)gridDim.x * blockDim.x) {
        if (!flag[i]) continue;
        const int o = pos[i];
        vox[o] = (int32_t)i;
        if (key) key[o] = lab[i];
    }
}

// length class of a row of the full set, longest first: 0..4 = more than 1024 / 512 / 256 / 128 / 64 entries (whole warp
// per row; the classes keep the static round-robin balanced), 5 = 33..64 (16 lanes per row), 6 = 17..32 (8 lanes),
// 7 = at most 16 (4 lanes)
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

// rows of a single-row (R = 1) set: entries = the row's non-zeros, padded to a multiple of 4
__global__ void k_fill_rows1(const int32_t* vox, const long long* ptr, long long n, int32_t* len, int32_t* ulen, long long* len64) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n; a += (long long)gridDim.x * blockDim.x) {
        const long long i = vox[a];
        const long long m = ptr[i + 1] - ptr[i];
        len[a] = (int32_t)((m + 3) & ~3LL);
        ulen[a] = (int32_t)m;
        len64[a] = (m + 3) & ~3LL;
    }
}

// Storage order inside a block row (or a transposed run) of Le entries (a multiple of C): every chunk of n <= 32 C entries
// (q = n / C lanes) is interleaved so that entry position C t + j of the chunk holds the chunk's logical entry t + q j.  A
// lane's 128-bit value load then yields the values of entries t, t + q, ..., and the j-th gather instruction of the warp
// covers q CONSECUTIVE entries: few cache lines of the gathered vector per instruction.  (C = 4: chunks of 128 entries.)
__host__ __device__ __forceinline__ long long perm_pos(long long e, long long Le, int C) {
    const int ce = 32 * C;
    const long long cb = e / ce * ce;
    const long long rem = Le - cb;
    const int n = rem < ce ? (int)rem : ce, q = n / C, r = (int)(e - cb);
    return cb + (long long)C * (r % q) + r / q;
}

__device__ __forceinline__ void st_col(int32_t* c32, uint16_t* c16, long long i, int v) { if (c16) c16[i] = (uint16_t)v; else c32[i] = v; }
__device__ __forceinline__ int ld_col(const int32_t* c32, const uint16_t* c16, long long i) { return c16 ? (int)c16[i] : c32[i]; }

// R = 1: copy the rows into the padded arrays (warp per row); padding stays {col 0, value 0}
__global__ void k_copy_rows1(long long n, const int32_t* vox, const long long* start, const long long* ptr, const int32_t* cU,
                             const float* uD, const float* uL, int32_t* col, uint16_t* col16, float* vD, float* vL) {
    const int lane = threadIdx.x & 31;
    const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long r = w0; r < n; r += nw) {
        const long long i = vox[r], b = ptr[i], e = ptr[i + 1], o = start[r];
        const long long Lp = (e - b + 3) & ~3LL;
        for (long long p = b + lane; p < e; p += 32) {
            const long long m = o + perm_pos(p - b, Lp, 4);
            st_col(col, col16, m, cU[p]);
            vD[m] = uD[p];
            vL[m] = uL[p];
        }
    }
}

// ---- block rows of the labelled set
// padded row index of the a-th labelled row (rows sorted by structure): a + shift[structure]; the other rows stay padding
__global__ void k_place_rows(long long n_act, const int32_t* vox_s, const int32_t* lab_s, const long long* shift, const long long* ptr,
                             int32_t* vox, int16_t* rseg, int32_t* rlen) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n_act; a += (long long)gridDim.x * blockDim.x) {
        const int sg = lab_s[a] - 1;
        const long long pa = a + shift[sg];
        const long long i = vox_s[a];
        vox[pa] = (int32_t)i;
        rseg[pa] = (int16_t)sg;
        rlen[pa] = (int32_t)(ptr[i + 1] - ptr[i]);
    }
}

// Union of the column patterns of the R rows of every block row (thread per block row: an R-way merge of sorted rows).
// COUNT: entries of the union.  FILL: the index and the R values per matrix of every entry (0 where a row has no entry).
template <int R, bool FILL>
__global__ void k_block_union(long long n_blk, const int32_t* __restrict__ vox, const long long* __restrict__ ptr,
                              const int32_t* __restrict__ cU, const float* __restrict__ uD, const float* __restrict__ uL,
                              long long* __restrict__ ecount,                                       // COUNT
                              const long long* __restrict__ start, const int32_t* __restrict__ len,  // FILL
                              int32_t* __restrict__ col, uint16_t* __restrict__ col16, float* __restrict__ vD, float* __restrict__ vL) {
    constexpr int C = 4 / R;
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < n_blk; b += (long long)gridDim.x * blockDim.x) {
        long long p[R], pe[R];
#pragma unroll
        for (int k = 0; k < R; ++k) {
            const int v = vox[b * R + k];
            p[k] = v >= 0 ? ptr[v] : 0;
            pe[k] = v >= 0 ? ptr[v + 1] : 0;
        }
        const long long o = FILL ? start[b] : 0;
        const long long Le = FILL ? len[b] : 0;
        long long e = 0;
        while (true) {
            int m = INT32_MAX;
#pragma unroll
            for (int k = 0; k < R; ++k) if (p[k] < pe[k]) { const int c = cU[p[k]]; m = c < m ? c : m; }
            if (m == INT32_MAX) break;
            if (FILL) {
                const long long pos = o + perm_pos(e, Le, C);
                st_col(col, col16, pos, m);
#pragma unroll
                for (int k = 0; k < R; ++k) {
                    const bool has = p[k] < pe[k] && cU[p[k]] == m;
                    vD[pos * R + k] = has ? uD[p[k]] : 0.f;
                    vL[pos * R + k] = has ? uL[p[k]] : 0.f;
                    if (has) ++p[k];
                }
            } else {
#pragma unroll
                for (int k = 0; k < R; ++k) if (p[k] < pe[k] && cU[p[k]] == m) ++p[k];
            }
            ++e;
        }
        if (!FILL) ecount[b] = e;
    }
}

// per block row: structure, real rows, padded length
__global__ void k_block_meta(long long n_blk, int R, const int16_t* rseg, const long long* ecount, int32_t* seg, int32_t* nreal,
                             int32_t* ulen, int32_t* len, long long* len64) {
    const int C = 4 / R;
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < n_blk; b += (long long)gridDim.x * blockDim.x) {
        int nr = 0;
        for (int k = 0; k < R; ++k) nr += rseg[b * R + k] >= 0;
        seg[b] = rseg[b * R];                      // row 0 of a block is always real
        nreal[b] = nr;
        const long long e = ecount[b], pl = (e + C - 1) / C * C;
        ulen[b] = (int32_t)e;
        len[b] = (int32_t)pl;
        len64[b] = pl;
    }
}

// squared norms of D_i, L_i and L_i - LETmax D_i in fp64 (warp per block row of the labelled set)
__global__ void k_norms(long long n_blk, int R, const long long* start, const int32_t* len, const int32_t* seg, const float* vD,
                        const float* vL, const StructInfo* tab, double* nD, double* nL, double* nT) {
    const int lane = threadIdx.x & 31;
    const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long b = w0; b < n_blk; b += nw) {
        const long long s = start[b];
        const int L = len[b];
        const StructInfo& T = tab[seg[b]];
        const double tm = (T.flags & F_LETD) ? T.letd_max : 0.0;
        for (int k = 0; k < R; ++k) {
            double a = 0.0, bb = 0.0, c = 0.0;
            for (int p = lane; p < L; p += 32) {
                const double dv = (double)vD[(s + p) * R + k], lv = (double)vL[(s + p) * R + k];
                a = fma(dv, dv, a);
                bb = fma(lv, lv, bb);
                const double t = lv - tm * dv;
                c = fma(t, t, c);
            }
            a = warp_sum(a); bb = warp_sum(bb); c = warp_sum(c);
            if (lane == 0) { nD[b * R + k] = a; nL[b * R + k] = bb; nT[b * R + k] = (T.flags & F_LETD) ? c : 0.0; }
        }
    }
}

// integer bookkeeping per structure (atomics on integers: order-independent result)
__global__ void k_count_sets(long long n_rows, const int16_t* rseg, const int32_t* rlen, const double* nD, const double* nL,
                             const double* nT, StructInfo* tab) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n_rows; a += (long long)gridDim.x * blockDim.x) {
        if (rseg[a] < 0) continue;
        StructInfo& T = tab[rseg[a]];
        const int f = T.flags;
        unsigned long long sets = 0, part = 0;
        if (f & F_DOSE_SLAB) { ++sets; part += nD[a] > 0.0; if (nD[a] > 0.0) atomicAdd(&T.part_kind[0], 1ULL); }
        if (f & F_DL_SLAB) { ++sets; part += nL[a] > 0.0; if (nL[a] > 0.0) atomicAdd(&T.part_kind[1], 1ULL); }
        if (f & F_LETD) { ++sets; part += nT[a] > 0.0; if (nT[a] > 0.0) atomicAdd(&T.part_kind[2], 1ULL); }
        atomicAdd(&T.n_sets, sets);
        atomicAdd(&T.part, part);
        atomicAdd(&T.n_zero, sets - part);
        atomicAdd(&T.rows, 1ULL);
        atomicAdd(&T.nnz, (unsigned long long)rlen[a]);
    }
}
// per-voxel LETd limits: |L_i - LETmax_i D_i|^2 of every row of a structure with an LETd limit (warp per block row)
__global__ void k_norms_letd(long long n_blk, int R, const long long* start, const int32_t* len, const int32_t* seg, const float* vD,
                             const float* vL, const StructInfo* tab, const double* tmax_row, double* nT) {
    const int lane = threadIdx.x & 31;
    const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long b = w0; b < n_blk; b += nw) {
        const StructInfo& T = tab[seg[b]];
        if (!(T.flags & F_LETD)) continue;
        const long long s = start[b];
        const int L = len[b];
        for (int k = 0; k < R; ++k) {
            const double tm = tmax_row ? tmax_row[b * R + k] : T.letd_max;
            double c = 0.0;
            for (int p = lane; p < L; p += 32) {
                const double t = (double)vL[(s + p) * R + k] - tm * (double)vD[(s + p) * R + k];
                c = fma(t, t, c);
            }
            c = warp_sum(c);
            if (lane == 0) nT[b * R + k] = c;
        }
    }
}
__global__ void k_reset_set_counts(StructInfo* tab, int n) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) { tab[s].part = 0; tab[s].n_sets = 0; tab[s].n_zero = 0; tab[s].part_kind[0] = tab[s].part_kind[1] = tab[s].part_kind[2] = 0; }
}
// the set bookkeeping of k_count_sets without the row / non-zero counts
__global__ void k_recount_sets(long long n_rows, const int16_t* rseg, const double* nD, const double* nL, const double* nT, StructInfo* tab) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n_rows; a += (long long)gridDim.x * blockDim.x) {
        if (rseg[a] < 0) continue;
        StructInfo& T = tab[rseg[a]];
        const int f = T.flags;
        unsigned long long sets = 0, part = 0;
        if (f & F_DOSE_SLAB) { ++sets; part += nD[a] > 0.0; if (nD[a] > 0.0) atomicAdd(&T.part_kind[0], 1ULL); }
        if (f & F_DL_SLAB) { ++sets; part += nL[a] > 0.0; if (nL[a] > 0.0) atomicAdd(&T.part_kind[1], 1ULL); }
        if (f & F_LETD) { ++sets; part += nT[a] > 0.0; if (nT[a] > 0.0) atomicAdd(&T.part_kind[2], 1ULL); }
        atomicAdd(&T.n_sets, sets);
        atomicAdd(&T.part, part);
        atomicAdd(&T.n_zero, sets - part);
    }
}
__global__ void k_count_entries(long long n_blk, const int32_t* seg, const int32_t* ulen, StructInfo* tab) {
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < n_blk; b += (long long)gridDim.x * blockDim.x)
        atomicAdd(&tab[seg[b]].entries, (unsigned long long)ulen[b]);
}
__global__ void k_label_hist(long long n, const int32_t* lab_s, unsigned long long* hist) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n; a += (long long)gridDim.x * blockDim.x)
        atomicAdd(hist + (lab_s[a] - 1), 1ULL);
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

// ---- transposition of a row set (entries = (block row, column) pairs with R values per matrix)
// key of an entry = ((segment * S + spot) * H + group) with group = block row >> 16 (H = 1: no groups)
__global__ void k_tr_keys(long long n, int C, const long long* start, const int32_t* len, const int32_t* ulen, const int32_t* seg,
                          const long long* off, const int32_t* col, const uint16_t* col16, long long S, int H, uint32_t* keys,
                          uint32_t* vals) {
    const int lane = threadIdx.x & 31;
    const long long w0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long r = w0; r < n; r += nw) {
        const long long s = start[r], o = off[r];
        const int L = ulen[r], Lp = len[r];
        const int sg = seg ? seg[r] : 0;
        for (int p = lane; p < L; p += 32) {
            keys[o + p] = ((uint32_t)sg * (uint32_t)S + (uint32_t)ld_col(col, col16, s + perm_pos(p, Lp, C))) * (uint32_t)H + (H > 1 ? (uint32_t)(r >> 16) : 0u);
            vals[o + p] = (uint32_t)(o + p);
        }
    }
}
// ustart[k] = first sorted position with key >= k, k = 0..K
__global__ void k_tr_bounds(const uint32_t* keys, long long E, long long K, long long* ustart) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k <= K; k += (long long)gridDim.x * blockDim.x) {
        long long lo = 0, hi = E;
        while (lo < hi) { const long long mid = (lo + hi) >> 1; if ((long long)keys[mid] < k) lo = mid + 1; else hi = mid; }
        ustart[k] = lo;
    }
}
__global__ void k_tr_pcount(const long long* ustart, long long K, int C, long long* pcount) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < K; k += (long long)gridDim.x * blockDim.x)
        pcount[k] = (ustart[k + 1] - ustart[k] + C - 1) / C * C;
}
__global__ void k_tr_fill(const uint32_t* keys, const uint32_t* vals, long long E, int R, const long long* ustart, const long long* t_ptr,
                          const long long* off, long long n_rows, const long long* start, const int32_t* len, const float* vD,
                          const float* vL, int32_t* t_col, uint16_t* t_col16, float* tD, float* tL) {
    const int C = 4 / R;
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < E; r += (long long)gridDim.x * blockDim.x) {
        const long long k = keys[r], e = vals[r];
        // block row a with off[a] <= e < off[a+1]
        long long lo = 0, hi = n_rows;
        while (lo < hi) { const long long mid = (lo + hi) >> 1; if (off[mid + 1] <= e) lo = mid + 1; else hi = mid; }
        const long long a = lo, p = start[a] + perm_pos(e - off[a], len[a], C);
        const long long dst = t_ptr[k] + perm_pos(r - ustart[k], t_ptr[k + 1] - t_ptr[k], C);
        if (t_col16) t_col16[dst] = (uint16_t)(a & 0xFFFF); else t_col[dst] = (int32_t)a;
        for (int kk = 0; kk < R; ++kk) {
            tD[dst * R + kk] = vD[p * R + kk];
            tL[dst * R + kk] = vL[p * R + kk];
        }
    }
}
// {start, len, seg, real rows} -> the 16-byte item the forward kernel reads (start / len in values per matrix)
__global__ void k_pack_items(long long n, int R, const long long* start, const int32_t* len, const int32_t* seg, const int32_t* nreal,
                             Item* items) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        Item it;
        it.start = start[i] * R; it.len = len[i] * R; it.seg = (seg ? seg[i] : 0) | ((nreal ? nreal[i] : 1) << 8);
        items[i] = it;
    }
}
// items per (spot, segment, group) run: ceil(values / TR_ITEM_MAX)
__global__ void k_tr_item_count(const long long* t_ptr, long long K, int R, int item_max, long long* cnt) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < K; k += (long long)gridDim.x * blockDim.x)
        cnt[k] = ((t_ptr[k + 1] - t_ptr[k]) * R + item_max - 1) / item_max;
}
// the same counts in spot-major order (the order of a spot's partial-sum slots)
__global__ void k_tr_item_count_sm(const long long* cnt, long long S, int n_seg, int H, long long* cnt_sm) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < S * n_seg * H; k += (long long)gridDim.x * blockDim.x) {
        const long long hi = k % H, js = k / H, j = js % S, sg = js / S;
        cnt_sm[(j * n_seg + sg) * H + hi] = cnt[k];
    }
}
// item.seg = segment | (group << 8): the kernel adds group << 16 to the 16-bit block-row indices
__global__ void k_tr_item_fill(const long long* t_ptr, const long long* ibase, const long long* sbase, long long S, int n_seg, int H, int R,
                               int item_max, Item* items, int32_t* item_slot) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < S * n_seg * H; k += (long long)gridDim.x * blockDim.x) {
        const long long b = t_ptr[k] * R, e = t_ptr[k + 1] * R;          // in values per matrix
        const long long hi = k % H, js = k / H, j = js % S, sg0 = js / S;
        const long long sg = sg0 | (hi << 8);
        long long i = ibase[k], slot = sbase[(j * n_seg + sg0) * H + hi];
        for (long long p = b; p < e; p += item_max, ++i, ++slot) {
            Item it;
            it.start = p; it.len = (int32_t)((e - p) < item_max ? (e - p) : item_max); it.seg = (int32_t)sg;
            items[i] = it;
            item_slot[i] = (int32_t)slot;
        }
    }
}
// longest-first execution order: key = length class (256-value bins, longest = 0); a stable sort keeps the
// (structure, spot) order inside a class
__global__ void k_tr_item_key(const Item* items, long long n, int item_max, uint32_t* key, uint32_t* idx) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        key[i] = (uint32_t)((item_max - items[i].len) / 256);
        idx[i] = (uint32_t)i;
    }
}
__global__ void k_tr_item_key_seg(const Item* items, long long n, int item_max, uint32_t* key, uint32_t* idx, unsigned long long* hist) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const uint32_t sg = (uint32_t)(items[i].seg & 0xFF);
        key[i] = sg * 16u + (uint32_t)((item_max - items[i].len) / 256);
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
// execution order of the forward items: longest first (stable: list order among equal lengths)
__global__ void k_item_len_key(const Item* items, long long n, uint32_t* key, uint32_t* idx) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        key[i] = 0xFFFFFFFFu - (uint32_t)items[i].len;
        idx[i] = (uint32_t)i;
    }
}
__global__ void k_item_gather(const uint32_t* idx, long long n, const Item* items, Item* items_x, int32_t* item_blk) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        items_x[i] = items[idx[i]];
        item_blk[i] = (int32_t)idx[i];
    }
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

// temporaries of a create-time routine: freed when the routine returns, whatever the path
struct TmpPool {
    std::vector<void*> v;
    ~TmpPool() { for (void* p : v) cudaFree(p); }
    template <class T>
    int get(T** p, size_t n) {
        *p = nullptr;
        CK(cudaMalloc((void**)p, (n ? n : 1) * sizeof(T)));
        v.push_back((void*)*p);
        return FREDOPT_OK;
    }
};

int build_transpose(fredopt_plan* P, RowSet& R) {
    cudaStream_t st = P->stream;
    const long long n = R.n, S = P->S;
    const int RB = R.R, C = 4 / RB;
    TmpPool T;
    // 16-bit block-row indices: cut every (segment, spot) run where the index crosses a multiple of 65536
    int H = (int)((n + 65535) >> 16);
    if (H < 1) H = 1;
    const bool idx16 = R.n_seg < 256 && H < (1 << 23) && (double)S * R.n_seg * H < 4.0e9 && !P->force_idx32;
    if (!idx16) H = 1;
    R.t_H = H;
    const long long K = S * R.n_seg * H;
    // offsets of the block rows in the enumeration of the (unpadded) entries
    long long *len64 = nullptr, *off = nullptr;
    CKR(T.get(&len64, (size_t)n + 1)); CKR(T.get(&off, (size_t)n + 2));
    CK(cudaMemsetAsync(len64, 0, (n + 1) * sizeof(long long), st));
    if (n) k_i32_to_i64<<<grid_for(n, 256, 4096), 256, 0, st>>>(R.ulen, len64, n);
    CKR(scan_exclusive(P, len64, off, n + 1));
    long long E = 0;
    CK(cudaMemcpyAsync(&E, off + n, sizeof(long long), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    R.entries = E;
    if (E >= (1LL << 32) || K >= (1LL << 32)) return FREDOPT_INVALID_ARG;
    uint32_t *keys = nullptr, *vals = nullptr, *keys2 = nullptr, *vals2 = nullptr;
    long long *ustart = nullptr, *pcount = nullptr;
    const size_t En = E ? (size_t)E : 1;
    CKR(T.get(&keys, En)); CKR(T.get(&vals, En)); CKR(T.get(&keys2, En)); CKR(T.get(&vals2, En));
    CKR(T.get(&ustart, (size_t)K + 2)); CKR(T.get(&pcount, (size_t)K + 2));
    if (n) k_tr_keys<<<grid_for(n * 32, 256, 1 << 16), 256, 0, st>>>(n, C, R.start, R.len, R.ulen, R.seg, off, R.col, R.col16, S, H, keys, vals);
    int bits = 1;
    while ((1LL << bits) < K) ++bits;
    {
        size_t tb = 0;
        void* tmp = nullptr;
        CK(cub::DeviceRadixSort::SortPairs(nullptr, tb, keys, keys2, vals, vals2, E, 0, bits, st));
        CKR(T.get((char**)&tmp, tb));
        CK(cub::DeviceRadixSort::SortPairs(tmp, tb, keys, keys2, vals, vals2, E, 0, bits, st));   // stable: list order kept inside a key
    }
    k_tr_bounds<<<grid_for(K + 1, 256, 4096), 256, 0, st>>>(keys2, E, K, ustart);
    CK(cudaMemsetAsync(pcount, 0, (K + 2) * sizeof(long long), st));
    k_tr_pcount<<<grid_for(K, 256, 4096), 256, 0, st>>>(ustart, K, C, pcount);
    CK(cudaGetLastError());
    CKR(dmalloc(P, &R.t_ptr, (size_t)K + 2));
    CKR(scan_exclusive(P, pcount, R.t_ptr, K + 1));
    CK(cudaMemcpyAsync(&R.t_entries_padded, R.t_ptr + K, sizeof(long long), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    const size_t Tn = R.t_entries_padded ? (size_t)R.t_entries_padded : 4;
    if (idx16) CKR(dmalloc(P, &R.t_col16, Tn + IDX_SLACK)); else CKR(dmalloc(P, &R.t_col, Tn + IDX_SLACK));   // slack: see IDX_SLACK
    CKR(dmalloc(P, &R.t_valD, Tn * RB)); CKR(dmalloc(P, &R.t_valL, Tn * RB));
    if (idx16) CK(cudaMemsetAsync(R.t_col16, 0, (Tn + IDX_SLACK) * 2, st)); else CK(cudaMemsetAsync(R.t_col, 0, (Tn + IDX_SLACK) * 4, st));
    CK(cudaMemsetAsync(R.t_valD, 0, Tn * RB * 4, st));
    CK(cudaMemsetAsync(R.t_valL, 0, Tn * RB * 4, st));
    if (E) k_tr_fill<<<grid_for(E, 256, 1 << 16), 256, 0, st>>>(keys2, vals2, E, RB, ustart, R.t_ptr, off, n, R.start, R.len, R.valD, R.valL,
                                                             R.t_col, R.t_col16, R.t_valD, R.t_valL);
    CK(cudaGetLastError());
    // ---- work items: every (segment, spot, group) run cut into pieces of at most TR_ITEM_MAX values, in run order
    //      (neighbouring items = neighbouring spots of one structure: overlapping voxel footprints share L1 lines)
    CK(cudaMemsetAsync(pcount, 0, (K + 2) * sizeof(long long), st));
    // Items of 3 072 values on large plans: 24 chunks are whole trips for both trip sizes (4 x 6 and 6 x 4 chunks), so no item ends on
    // a ragged trip (configs[3] +1.4 %, configs[2] +1.7 %); small plans keep 2 048 (configs[1] -5 % with 3 072: fewer items than warps).
    const int item_max = (&R == &P->act && R.nnz >= 50000000LL) ? 3072 : TR_ITEM_MAX;
    static_assert(3072 % 256 == 0 && 3072 / 256 < 16, "length-class keys");
    k_tr_item_count<<<grid_for(K, 256, 4096), 256, 0, st>>>(R.t_ptr, K, RB, item_max, pcount);
    long long* cnt_sm = nullptr;
    CKR(T.get(&cnt_sm, (size_t)K + 2));
    CKR(dmalloc(P, &R.t_slot_ptr, (size_t)K + 2));       // kept: slot ranges per (spot, structure, group) for the block-sequential sweep
    long long* sbase = R.t_slot_ptr;
    CK(cudaMemsetAsync(cnt_sm, 0, (K + 2) * sizeof(long long), st));
    k_tr_item_count_sm<<<grid_for(K, 256, 4096), 256, 0, st>>>(pcount, S, R.n_seg, H, cnt_sm);
    CKR(scan_exclusive(P, pcount, ustart, K + 1));       // ustart now = first item of each run (execution order)
    CKR(scan_exclusive(P, cnt_sm, sbase, K + 1));        // first partial-sum slot of each (spot, segment, group)
    CK(cudaMemcpyAsync(&R.t_n_items, ustart + K, sizeof(long long), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    CKR(dmalloc(P, &R.t_items, (size_t)R.t_n_items)); CKR(dmalloc(P, &R.t_item_slot, (size_t)R.t_n_items));
    CKR(dmalloc(P, &R.t_item_ptr, (size_t)S + 1)); CKR(dmalloc(P, &R.t_partial, (size_t)R.t_n_items));
    k_tr_item_fill<<<grid_for(K, 256, 4096), 256, 0, st>>>(R.t_ptr, ustart, sbase, S, R.n_seg, H, RB, item_max, R.t_items, R.t_item_slot);
    k_tr_item_ptr<<<grid_for(S + 1, 256, 4096), 256, 0, st>>>(sbase, S, (long long)R.n_seg * H, R.t_item_ptr);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(st));
    // ---- the same items grouped by structure, longest first inside a structure (block-sequential AMS)
    R.t_seg_item_begin.assign((size_t)R.n_seg + 1, 0);
    if (R.t_n_items > 0) {
        const long long ni = R.t_n_items;
        uint32_t *ik = nullptr, *ik2 = nullptr, *ii = nullptr, *ii2 = nullptr;
        unsigned long long* hist = nullptr;
        CKR(T.get(&ik, (size_t)ni)); CKR(T.get(&ik2, (size_t)ni)); CKR(T.get(&ii, (size_t)ni)); CKR(T.get(&ii2, (size_t)ni));
        CKR(T.get(&hist, 256));
        CK(cudaMemsetAsync(hist, 0, 256 * 8, st));
        CKR(dmalloc(P, &R.t_items_seg, (size_t)ni)); CKR(dmalloc(P, &R.t_slot_seg, (size_t)ni));
        k_tr_item_key_seg<<<grid_for(ni, 256, 4096), 256, 0, st>>>(R.t_items, ni, item_max, ik, ii, hist);
        size_t sb = 0;
        void* stmp = nullptr;
        CK(cub::DeviceRadixSort::SortPairs(nullptr, sb, ik, ik2, ii, ii2, ni, 0, 12, st));
        CKR(T.get((char**)&stmp, sb));
        CK(cub::DeviceRadixSort::SortPairs(stmp, sb, ik, ik2, ii, ii2, ni, 0, 12, st));
        k_tr_item_permute<<<grid_for(ni, 256, 4096), 256, 0, st>>>(ii2, ni, R.t_items, R.t_item_slot, R.t_items_seg, R.t_slot_seg);
        unsigned long long hh[256];
        CK(cudaMemcpyAsync(hh, hist, 256 * 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        for (int sg = 0; sg < R.n_seg; ++sg) R.t_seg_item_begin[sg + 1] = R.t_seg_item_begin[sg] + (long long)hh[sg];
    }
    // ---- the items in run order (= storage order) are kept beside the longest-first list
    if (R.t_n_items > 0) {
        CKR(dmalloc(P, &R.t_items_run, (size_t)R.t_n_items)); CKR(dmalloc(P, &R.t_slot_run, (size_t)R.t_n_items));
        CK(cudaMemcpyAsync(R.t_items_run, R.t_items, R.t_n_items * sizeof(Item), cudaMemcpyDeviceToDevice, st));
        CK(cudaMemcpyAsync(R.t_slot_run, R.t_item_slot, R.t_n_items * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    }
    // ---- longest items first: with the static round-robin mapping every round of the grid then holds items of
    //      one length class, so the warps stay balanced to within one class width per round
    if (R.t_n_items > 1) {
        const long long ni = R.t_n_items;
        uint32_t *ik = nullptr, *ik2 = nullptr, *ii = nullptr, *ii2 = nullptr;
        Item* it2 = nullptr; int32_t* js2 = nullptr;
        CKR(T.get(&ik, (size_t)ni)); CKR(T.get(&ik2, (size_t)ni)); CKR(T.get(&ii, (size_t)ni)); CKR(T.get(&ii2, (size_t)ni));
        CKR(T.get(&it2, (size_t)ni)); CKR(T.get(&js2, (size_t)ni));
        k_tr_item_key<<<grid_for(ni, 256, 4096), 256, 0, st>>>(R.t_items, ni, item_max, ik, ii);
        size_t sb = 0;
        void* stmp = nullptr;
        CK(cub::DeviceRadixSort::SortPairs(nullptr, sb, ik, ik2, ii, ii2, ni, 0, 4, st));
        CKR(T.get((char**)&stmp, sb));
        CK(cub::DeviceRadixSort::SortPairs(stmp, sb, ik, ik2, ii, ii2, ni, 0, 4, st));
        k_tr_item_permute<<<grid_for(ni, 256, 4096), 256, 0, st>>>(ii2, ni, R.t_items, R.t_item_slot, it2, js2);
        CK(cudaMemcpyAsync(R.t_items, it2, ni * sizeof(Item), cudaMemcpyDeviceToDevice, st));
        CK(cudaMemcpyAsync(R.t_item_slot, js2, ni * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
        CK(cudaStreamSynchronize(st));
    }
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(st));
    R.t_built = true;
    return FREDOPT_OK;
}

// Sharded plans: the set counts of the WHOLE plan (participating / declared / zero-norm sets per structure and kind) are the
// sums of the ranks' local counts -> W, w^.  Call right after a local count.
static int reduce_set_counts(fredopt_plan* P) {
    // the set counts of the WHOLE plan: participating / declared / zero-norm sets per structure and kind -> W, w^
    const int ns = P->n_struct;
    std::vector<double> h((size_t)ns * 6 + 1, 0.0);
    CK(cudaMemcpyAsync(P->h_tab.data(), P->tab, sizeof(StructInfo) * P->max_seg, cudaMemcpyDeviceToHost, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    for (int s = 0; s < ns; ++s) {
        const StructInfo& T = P->h_tab[s];
        h[s * 6 + 0] = (double)T.part; h[s * 6 + 1] = (double)T.n_sets; h[s * 6 + 2] = (double)T.n_zero;
        h[s * 6 + 3] = (double)T.part_kind[0]; h[s * 6 + 4] = (double)T.part_kind[1]; h[s * 6 + 5] = (double)T.part_kind[2];
    }
    double* d = nullptr;
    CK(cudaMalloc((void**)&d, h.size() * 8));
    cudaError_t e = cudaMemcpyAsync(d, h.data(), h.size() * 8, cudaMemcpyHostToDevice, P->stream);
    int rc = e == cudaSuccess ? reduce_call(P, d, (long long)h.size()) : FREDOPT_CUDA_ERROR;
    if (rc == FREDOPT_OK) e = cudaMemcpyAsync(h.data(), d, h.size() * 8, cudaMemcpyDeviceToHost, P->stream);
    cudaError_t e2 = cudaStreamSynchronize(P->stream);
    cudaFree(d);
    if (rc != FREDOPT_OK) return rc;
    CK(e); CK(e2);
    for (int s = 0; s < ns; ++s) {
        StructInfo& T = P->h_tab[s];
        T.part = (unsigned long long)h[s * 6 + 0]; T.n_sets = (unsigned long long)h[s * 6 + 1]; T.n_zero = (unsigned long long)h[s * 6 + 2];
        T.part_kind[0] = (unsigned long long)h[s * 6 + 3]; T.part_kind[1] = (unsigned long long)h[s * 6 + 4]; T.part_kind[2] = (unsigned long long)h[s * 6 + 5];
    }
    CK(cudaMemcpyAsync(P->tab, P->h_tab.data(), sizeof(StructInfo) * P->max_seg, cudaMemcpyHostToDevice, P->stream));
    k_finish_tables<<<1, 1, 0, P->stream>>>(P->tab, P->n_struct, P->st, P->mode_union, P->mode_con, P->mode_cost, P->mode_fixed, P->max_seg);
    CK(cudaMemcpyAsync(P->h_tab.data(), P->tab, sizeof(StructInfo) * P->max_seg, cudaMemcpyDeviceToHost, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    CK(cudaGetLastError());
    return FREDOPT_OK;
}

int recount_sets(fredopt_plan* P, bool letd_norms) {
    cudaStream_t st = P->stream;
    const RowSet& A = P->act;
    const int ns = P->max_seg;
    if (A.n && letd_norms)
        k_norms_letd<<<grid_for(A.n * 32, 256, 1 << 16), 256, 0, st>>>(A.n, A.R, A.start, A.len, A.seg, A.valD, A.valL, P->tab, P->vb.f[VB_LETD_MAX], P->nT);
    k_reset_set_counts<<<1, 256, 0, st>>>(P->tab, P->n_struct);
    if (A.n_rows) k_recount_sets<<<grid_for(A.n_rows, 256, 4096), 256, 0, st>>>(A.n_rows, A.rseg, P->nD, P->nL, P->nT, P->tab);
    k_finish_tables<<<1, 1, 0, st>>>(P->tab, P->n_struct, P->st, P->mode_union, P->mode_con, P->mode_cost, P->mode_fixed, ns);
    CK(cudaMemcpyAsync(P->h_tab.data(), P->tab, sizeof(StructInfo) * ns, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    if (P->shard_world > 1 && P->reduce_fn) CKR(reduce_set_counts(P));
    return FREDOPT_OK;
}

// Bytes the method must move in one launch of a pass: per non-zero of a row 4 B for every value array the
// row's structure needs in that pass; per stored entry (one per block row and column of the union pattern) the stored index
// (2 B, or 4 B in the 32-bit form); 8 B per row offset; the fp64 vectors read / written once.  The zeros a block row stores
// where one of its rows has no entry are NOT counted (they show up as DRAM traffic above this figure).
static void compute_pass_bytes(fredopt_plan* P) {
    long long fwd_union = 0, tr_cost = 0, tr_con = 0, rows_union = 0, rows_con = 0, rows_cost = 0, con_values = 0;
    const int ibf = P->act.col16 ? 2 : 4, ibt = P->act.t_col16 ? 2 : 4;     // index bytes as stored
    for (int s = 0; s < P->n_struct; ++s) {
        const StructInfo& T = P->h_tab[s];
        const int f = T.flags;
        const int cost = ((f & F_DOSE_REF) ? 1 : 0) | ((f & F_DL_REF) ? 2 : 0);
        const int con = ((f & (F_DOSE_SLAB | F_LETD)) ? 1 : 0) | ((f & (F_DL_SLAB | F_LETD)) ? 2 : 0);
        const int vw = P->act.valD16 ? 2 : 4;                                   // value bytes as stored
        auto per = [&](int m, int ib) { return m ? (long long)T.entries * ib + (long long)T.nnz * vw * ((m & 1) + ((m >> 1) & 1)) : 0LL; };
        fwd_union += per(cost | con, ibf);
        tr_cost += per(cost, ibt);
        tr_con += per(con, ibt);
        con_values += (long long)T.nnz * vw * ((con & 1) + ((con >> 1) & 1));
        if (cost | con) rows_union += T.rows;
        if (con) rows_con += T.rows;
        if (cost) rows_cost += T.rows;
    }
    const long long S = P->S, VA = P->act.n_true;
    P->pass_bytes[FREDOPT_PASS_FORWARD_X] = fwd_union + rows_union * (8 + 16) + S * 8;
    P->pass_bytes[FREDOPT_PASS_FORWARD_G] = fwd_union + rows_union * (8 + 16) + S * 8;
    P->pass_bytes[FREDOPT_PASS_TRANSPOSE_G] = tr_cost + S * P->act.n_seg * 8 + rows_cost * 16 + S * 8;
    P->pass_bytes[FREDOPT_PASS_TRANSPOSE_B] = tr_con + S * P->act.n_seg * 8 + rows_con * 16 + S * 16;
    P->tr_con_value_bytes = con_values;
    P->pass_bytes[FREDOPT_PASS_SELECT] = S * 24;
    P->pass_bytes[FREDOPT_PASS_RESIDUAL] = VA * (4 + 8 * 9);
}

// ============================================================================================ API
extern "C" {

#ifdef FREDOPT_CHECKED
}   // extern "C"
#include <mutex>
static std::mutex g_chk_mu;
static std::vector<ChkRange> g_chk_host;
static unsigned long long g_chk_version = 0, g_chk_uploaded = ~0ull;
void chk_register(const void* p, size_t bytes) {
    std::lock_guard<std::mutex> lk(g_chk_mu);
    g_chk_host.push_back(ChkRange{(const char*)p, (const char*)p + bytes});
    ++g_chk_version;
}
void chk_unregister(const void* p) {
    std::lock_guard<std::mutex> lk(g_chk_mu);
    for (size_t i = 0; i < g_chk_host.size(); ++i)
        if (g_chk_host[i].b == (const char*)p) { g_chk_host[i] = g_chk_host.back(); g_chk_host.pop_back(); ++g_chk_version; break; }
}
void chk_upload_build(const ChkRange* h, int n) { chk_upload_tu(h, n); }
void chk_sync(cudaStream_t stream) {
    std::lock_guard<std::mutex> lk(g_chk_mu);
    if (g_chk_uploaded == g_chk_version) return;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (stream && cudaStreamIsCapturing(stream, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone) return;
    cudaDeviceSynchronize();
    const int n = (int)(g_chk_host.size() < (size_t)CHK_MAX ? g_chk_host.size() : (size_t)CHK_MAX);
    chk_upload_iterate(g_chk_host.data(), n); chk_upload_passes(g_chk_host.data(), n); chk_upload_build(g_chk_host.data(), n);
    cudaDeviceSynchronize();
    g_chk_uploaded = g_chk_version;
}
extern "C" {
#endif

void fredopt_destroy(fredopt_plan* P) {
    if (!P) return;
    cudaStreamSynchronize(P->stream);
    for (auto& ep : P->events) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
    for (auto& ep : P->event_pool) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
    for (int i = 0; i < 8; ++i) if (P->gexec[i]) cudaGraphExecDestroy(P->gexec[i]);
    for (void* p : P->allocs) { chk_unregister(p); cudaFree(p); }
    if (P->st_host) cudaFreeHost(P->st_host);
    for (int k = 0; k < VB_N; ++k) cudaFree(P->vb_buf[k]);
    if (P->owns_stream) cudaStreamDestroy(P->stream);
    delete P;
}

}  // extern "C"

// union-pattern entries of the labelled rows grouped R at a time (rows placed in `vox`, n_blk block rows)
template <int R>
static int count_union(fredopt_plan* P, long long n_blk, const int32_t* vox, const long long* pU, const int32_t* cU, long long* ecount,
                       long long* total) {
    if (n_blk) k_block_union<R, false><<<grid_for(n_blk, 128, 1 << 16), 128, 0, P->stream>>>(n_blk, vox, pU, cU, nullptr, nullptr, ecount, nullptr,
                                                                                       nullptr, nullptr, nullptr, nullptr, nullptr);
    size_t tb = 0;
    long long* dsum = nullptr;
    void* tmp = nullptr;
    TmpPool T;
    CKR(T.get(&dsum, 1));
    CK(cub::DeviceReduce::Sum(nullptr, tb, ecount, dsum, n_blk, P->stream));
    CKR(T.get((char**)&tmp, tb));
    CK(cub::DeviceReduce::Sum(tmp, tb, ecount, dsum, n_blk, P->stream));
    CK(cudaMemcpyAsync(total, dsum, 8, cudaMemcpyDeviceToHost, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    CK(cudaGetLastError());
    return FREDOPT_OK;
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
    TmpPool tmp;   // temporaries of this call
    auto to_dev = [&](const void* src, size_t bytes, const void** out) -> int {
        if (bytes == 0) { char* p; CKR(tmp.get(&p, 16)); *out = p; return FREDOPT_OK; }
        if (is_device_ptr(src)) { *out = src; return FREDOPT_OK; }
        char* p = nullptr;
        CKR(tmp.get(&p, bytes));
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
    CKR(tmp.get(&flag, 3));                                      // [0] invalid input, [1] patterns differ, [2] a value beyond the range of a half
    CK(cudaMemsetAsync(flag, 0, 3 * sizeof(int), st));
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
        CKR(tmp.get(&cnt, (size_t)V + 1)); CKR(tmp.get(&pu, (size_t)V + 2));
        CK(cudaMemsetAsync(cnt, 0, (V + 1) * 8, st));
        k_union_count<<<grid_for(V, 128, 1 << 16), 128, 0, st>>>(pD, cD, pL, cL, V, cnt);
        CKR(scan_exclusive(P, cnt, pu, V + 1));
        CK(cudaMemcpyAsync(&nnzU, pu + V, 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        int32_t* cu; float *ud, *ul;
        CKR(tmp.get(&cu, (size_t)nnzU)); CKR(tmp.get(&ud, (size_t)nnzU)); CKR(tmp.get(&ul, (size_t)nnzU));
        k_union_fill<<<grid_for(V, 128, 1 << 16), 128, 0, st>>>(pD, cD, vD, pL, cL, vL, V, pu, cu, ud, ul);
        pU = pu; cU = cu; uD = ud; uL = ul;
    }
    if (nnzU >= (1LL << 32)) return FREDOPT_INVALID_ARG;
    P->nnz = nnzU;
    const bool idx16 = S <= 65536 && !P->force_idx32;       // 16-bit column indices for the hot kernels
    // ---- non-empty list, labelled list
    int32_t *f_ne, *f_act, *pos_ne, *pos_act;
    CKR(tmp.get(&f_ne, (size_t)V + 1)); CKR(tmp.get(&f_act, (size_t)V + 1));
    CKR(tmp.get(&pos_ne, (size_t)V + 2)); CKR(tmp.get(&pos_act, (size_t)V + 2));
    CK(cudaMemsetAsync(f_ne, 0, (V + 1) * 4, st));
    CK(cudaMemsetAsync(f_act, 0, (V + 1) * 4, st));
    P->shard_begin = 0; P->shard_end = V;
    if (P->shard_world > 1) {      // the cuts are computed on the host from D's row offsets and the labels (every rank: the same cuts)
        std::vector<long long> hp((size_t)V + 1);
        std::vector<int32_t> hl((size_t)(V ? V : 1));
        CK(cudaMemcpyAsync(hp.data(), pD, (V + 1) * 8, cudaMemcpyDefault, st));
        CK(cudaMemcpyAsync(hl.data(), lab, V * 4, cudaMemcpyDefault, st));
        CK(cudaStreamSynchronize(st));
        int64_t b = 0, e = 0;
        CKR(fredopt_shard_range((const int64_t*)hp.data(), hl.data(), V, P->shard_rank, P->shard_world, &b, &e));
        P->shard_begin = b; P->shard_end = e;
    }
    if (V) k_row_lengths<<<grid_for(V, 256, 1 << 16), 256, 0, st>>>(pU, lab, V, P->shard_begin, P->shard_end, f_ne, f_act);
    CKR(scan_exclusive(P, f_ne, pos_ne, V + 1));
    CKR(scan_exclusive(P, f_act, pos_act, V + 1));
    int32_t n_ne = 0, n_act = 0;
    CK(cudaMemcpyAsync(&n_ne, pos_ne + V, 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(&n_act, pos_act + V, 4, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    // ---- full row set (R = 1): non-empty rows ordered by (length class, voxel) and stored in that order, so that short rows
    //      (entrance channels, few spots per voxel) are handled by sub-warps over contiguous memory
    RowSet& F = P->full;
    F.R = 1; F.n = n_ne; F.n_rows = n_ne; F.n_true = n_ne; F.n_seg = 1; F.nnz = nnzU; F.entries = nnzU;
    CKR(dmalloc(P, &F.vox, (size_t)n_ne)); CKR(dmalloc(P, &F.start, (size_t)n_ne + 1));
    CKR(dmalloc(P, &F.len, (size_t)n_ne)); CKR(dmalloc(P, &F.ulen, (size_t)n_ne)); CKR(dmalloc(P, &F.items, (size_t)n_ne));
    {
        TmpPool t2;
        int32_t *vox0, *key0, *key1;
        long long* flen64;
        unsigned long long* hist;
        CKR(t2.get(&vox0, (size_t)n_ne + 1)); CKR(t2.get(&key0, (size_t)n_ne + 1)); CKR(t2.get(&key1, (size_t)n_ne + 1));
        CKR(t2.get(&flen64, (size_t)n_ne + 1)); CKR(t2.get(&hist, N_LEN_CLASS));
        CK(cudaMemsetAsync(hist, 0, N_LEN_CLASS * 8, st));
        if (V) k_compact_rows<<<grid_for(V, 256, 1 << 16), 256, 0, st>>>(f_ne, pos_ne, lab, V, vox0, nullptr);
        if (n_ne) k_class_keys<<<grid_for(n_ne, 256, 1 << 16), 256, 0, st>>>(vox0, pU, n_ne, key0, hist);
        size_t tb = 0;
        CK(cub::DeviceRadixSort::SortPairs(nullptr, tb, key0, key1, vox0, F.vox, n_ne, 0, 3, st));
        char* ts; CKR(t2.get(&ts, tb));
        CK(cub::DeviceRadixSort::SortPairs(ts, tb, key0, key1, vox0, F.vox, n_ne, 0, 3, st));   // stable: voxel order inside a class
        CK(cudaMemsetAsync(flen64, 0, ((size_t)n_ne + 1) * 8, st));
        if (n_ne) k_fill_rows1<<<grid_for(n_ne, 256, 1 << 16), 256, 0, st>>>(F.vox, pU, n_ne, F.len, F.ulen, flen64);
        CKR(scan_exclusive(P, flen64, F.start, (long long)n_ne + 1));
        unsigned long long hh[N_LEN_CLASS];
        CK(cudaMemcpyAsync(hh, hist, N_LEN_CLASS * 8, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(&F.entries_padded, F.start + n_ne, 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        P->nnz_padded = F.entries_padded;
        P->full_class[0] = 0;
        for (int c = 0; c < N_LEN_CLASS; ++c) P->full_class[c + 1] = P->full_class[c] + (long long)hh[c];
        const size_t np = F.entries_padded ? (size_t)F.entries_padded : 4;
        if (idx16) { CKR(dmalloc(P, &F.col16, np + IDX_SLACK)); CK(cudaMemsetAsync(F.col16, 0, (np + IDX_SLACK) * 2, st)); }
        else { CKR(dmalloc(P, &F.col, np + IDX_SLACK)); CK(cudaMemsetAsync(F.col, 0, (np + IDX_SLACK) * 4, st)); }
        CKR(dmalloc(P, &F.valD, np)); CKR(dmalloc(P, &F.valL, np));
        CK(cudaMemsetAsync(F.valD, 0, np * 4, st)); CK(cudaMemsetAsync(F.valL, 0, np * 4, st));
        if (n_ne) {
            k_copy_rows1<<<grid_for((long long)n_ne * 32, 256, 1 << 16), 256, 0, st>>>(F.n, F.vox, F.start, pU, cU, uD, uL, F.col, F.col16, F.valD, F.valL);
            if (P->value_bits == 16) {
                k_round_to_half<<<P->sm_count * 8, 256, 0, st>>>(F.valD, np, flag + 2);
                k_round_to_half<<<P->sm_count * 8, 256, 0, st>>>(F.valL, np, flag + 2);
            }
            k_pack_items<<<grid_for(n_ne, 256, 4096), 256, 0, st>>>(n_ne, 1, F.start, F.len, nullptr, nullptr, F.items);
        }
        CK(cudaStreamSynchronize(st));
        CK(cudaGetLastError());
    }
    // ---- labelled row set, ordered by (label, voxel), as block rows of R consecutive rows of one structure with its own
    //      compact copy of the entries: the iteration streams contiguous arrays (no unconstrained rows in between)
    RowSet& A = P->act;
    const int ns = n_struct > 0 ? n_struct : 1;
    A.n_seg = ns; A.n_true = n_act;
    P->max_seg = ns;
    CKR(dmalloc(P, &P->tab, (size_t)ns));
    CK(cudaMemcpyAsync(P->tab, P->h_tab.data(), sizeof(StructInfo) * ns, cudaMemcpyHostToDevice, st));
    {
        TmpPool t2;
        int32_t *vox0, *key0, *lab_s, *vox_s;
        unsigned long long* hist;
        CKR(t2.get(&vox0, (size_t)n_act + 1)); CKR(t2.get(&key0, (size_t)n_act + 1)); CKR(t2.get(&lab_s, (size_t)n_act + 1));
        CKR(t2.get(&vox_s, (size_t)n_act + 1)); CKR(t2.get(&hist, (size_t)ns));
        CK(cudaMemsetAsync(hist, 0, (size_t)ns * 8, st));
        if (V) k_compact_rows<<<grid_for(V, 256, 1 << 16), 256, 0, st>>>(f_act, pos_act, lab, V, vox0, key0);
        int bits = 1;
        while ((1 << bits) <= n_struct) ++bits;
        size_t tb = 0;
        CK(cub::DeviceRadixSort::SortPairs(nullptr, tb, key0, lab_s, vox0, vox_s, n_act, 0, bits, st));
        char* ts; CKR(t2.get(&ts, tb));
        CK(cub::DeviceRadixSort::SortPairs(ts, tb, key0, lab_s, vox0, vox_s, n_act, 0, bits, st));
        if (n_act) k_label_hist<<<grid_for(n_act, 256, 4096), 256, 0, st>>>(n_act, lab_s, hist);
        std::vector<unsigned long long> hrows((size_t)ns, 0ULL);
        CK(cudaMemcpyAsync(hrows.data(), hist, (size_t)ns * 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        // rows of a structure padded to a multiple of R, so that no block row straddles two structures
        long long* shift_d; CKR(t2.get(&shift_d, (size_t)ns));
        std::vector<long long> shift((size_t)ns, 0);
        auto layout = [&](int R, long long* n_rows_out) {
            long long base = 0, base_pad = 0;
            P->row_base.assign((size_t)ns + 1, 0);
            for (int s = 0; s < ns; ++s) {
                P->row_base[s] = base_pad;
                shift[s] = base_pad - base;
                base += (long long)hrows[s];
                base_pad += ((long long)hrows[s] + R - 1) / R * R;
            }
            P->row_base[ns] = base_pad;
            *n_rows_out = base_pad;
        };
        int32_t *rlen = nullptr;
        long long* ecount = nullptr;
        auto place = [&](int R, long long* n_rows_out) -> int {      // A.vox / A.rseg / rlen for block height R
            layout(R, n_rows_out);
            const long long nr = *n_rows_out;
            CK(cudaMemcpyAsync(shift_d, shift.data(), (size_t)ns * 8, cudaMemcpyHostToDevice, st));
            CK(cudaMemsetAsync(A.vox, 0xFF, (size_t)(nr ? nr : 1) * 4, st));
            CK(cudaMemsetAsync(A.rseg, 0xFF, (size_t)(nr ? nr : 1) * 2, st));
            CK(cudaMemsetAsync(rlen, 0, (size_t)(nr ? nr : 1) * 4, st));
            if (n_act) k_place_rows<<<grid_for(n_act, 256, 4096), 256, 0, st>>>(n_act, vox_s, lab_s, shift_d, pU, A.vox, A.rseg, rlen);
            CK(cudaStreamSynchronize(st));          // `shift` is reused by the next call
            return FREDOPT_OK;
        };
        const size_t max_rows = (size_t)n_act + 4 * (size_t)ns + 4;
        CKR(dmalloc(P, &A.vox, max_rows)); CKR(dmalloc(P, &A.rseg, max_rows));
        CKR(t2.get(&rlen, max_rows)); CKR(t2.get(&ecount, max_rows));
        // block height: the one that stores the fewest bytes (an index per entry + R values); a forced value wins
        long long nnzA = 0;
        int Rb = P->block_rows_opt;
        {
            long long nr1 = 0;
            CKR(place(1, &nr1));
            CKR(count_union<1>(P, nr1, A.vox, pU, cU, ecount, &nnzA));
        }
        A.nnz = nnzA;
        if (Rb == 0) {
            const double ib = idx16 ? 2.0 : 4.0;
            double best = (double)nnzA * (4.0 + ib);
            Rb = 1;
            for (int R : {2, 4}) {
                long long nr = 0, ent = 0;
                CKR(place(R, &nr));
                if (R == 2) CKR(count_union<2>(P, nr / R, A.vox, pU, cU, ecount, &ent));
                else CKR(count_union<4>(P, nr / R, A.vox, pU, cU, ecount, &ent));
                const double bytes = (double)ent * (4.0 * R + ib);
                if (bytes < 0.97 * best) { best = bytes; Rb = R; }      // a taller block must save at least 3 %
            }
        }
        A.R = Rb;
        long long n_rows = 0;
        CKR(place(Rb, &n_rows));
        A.n_rows = n_rows;
        A.n = n_rows / Rb;
        const long long n_blk = A.n;
        long long ent = 0;
        if (Rb == 1) CKR(count_union<1>(P, n_blk, A.vox, pU, cU, ecount, &ent));
        else if (Rb == 2) CKR(count_union<2>(P, n_blk, A.vox, pU, cU, ecount, &ent));
        else CKR(count_union<4>(P, n_blk, A.vox, pU, cU, ecount, &ent));
        A.entries = ent;
        CKR(dmalloc(P, &A.start, (size_t)n_blk + 1)); CKR(dmalloc(P, &A.len, (size_t)n_blk)); CKR(dmalloc(P, &A.ulen, (size_t)n_blk));
        CKR(dmalloc(P, &A.seg, (size_t)n_blk)); CKR(dmalloc(P, &A.items, (size_t)n_blk));
        int32_t* nreal; long long* len64;
        CKR(t2.get(&nreal, (size_t)n_blk)); CKR(t2.get(&len64, (size_t)n_blk + 1));
        CK(cudaMemsetAsync(len64, 0, ((size_t)n_blk + 1) * 8, st));
        if (n_blk) k_block_meta<<<grid_for(n_blk, 256, 4096), 256, 0, st>>>(n_blk, Rb, A.rseg, ecount, A.seg, nreal, A.ulen, A.len, len64);
        CKR(scan_exclusive(P, len64, A.start, n_blk + 1));
        CK(cudaMemcpyAsync(&A.entries_padded, A.start + n_blk, 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        const size_t na = A.entries_padded ? (size_t)A.entries_padded : 4;
        if (idx16) { CKR(dmalloc(P, &A.col16, na + IDX_SLACK)); CK(cudaMemsetAsync(A.col16, 0, (na + IDX_SLACK) * 2, st)); }
        else { CKR(dmalloc(P, &A.col, na + IDX_SLACK)); CK(cudaMemsetAsync(A.col, 0, (na + IDX_SLACK) * 4, st)); }
        CKR(dmalloc(P, &A.valD, na * Rb)); CKR(dmalloc(P, &A.valL, na * Rb));
        CK(cudaMemsetAsync(A.valD, 0, na * Rb * 4, st)); CK(cudaMemsetAsync(A.valL, 0, na * Rb * 4, st));
        if (n_blk) {
            const int g = grid_for(n_blk, 128, 1 << 16);
            if (Rb == 1) k_block_union<1, true><<<g, 128, 0, st>>>(n_blk, A.vox, pU, cU, uD, uL, nullptr, A.start, A.len, A.col, A.col16, A.valD, A.valL);
            else if (Rb == 2) k_block_union<2, true><<<g, 128, 0, st>>>(n_blk, A.vox, pU, cU, uD, uL, nullptr, A.start, A.len, A.col, A.col16, A.valD, A.valL);
            else k_block_union<4, true><<<g, 128, 0, st>>>(n_blk, A.vox, pU, cU, uD, uL, nullptr, A.start, A.len, A.col, A.col16, A.valD, A.valL);
            if (P->value_bits == 16) {      // before the norms: everything that follows sees the rounded values
                k_round_to_half<<<P->sm_count * 8, 256, 0, st>>>(A.valD, na * Rb, flag + 2);
                k_round_to_half<<<P->sm_count * 8, 256, 0, st>>>(A.valL, na * Rb, flag + 2);
            }
            k_pack_items<<<grid_for(n_blk, 256, 4096), 256, 0, st>>>(n_blk, Rb, A.start, A.len, A.seg, nreal, A.items);
            // execution order of the whole-set passes: longest block rows first (the queue then ends with the short ones)
            uint32_t *ik, *ik2, *ii, *ii2;
            CKR(t2.get(&ik, (size_t)n_blk)); CKR(t2.get(&ik2, (size_t)n_blk)); CKR(t2.get(&ii, (size_t)n_blk)); CKR(t2.get(&ii2, (size_t)n_blk));
            CKR(dmalloc(P, &A.items_x, (size_t)n_blk)); CKR(dmalloc(P, &A.item_blk, (size_t)n_blk));
            k_item_len_key<<<grid_for(n_blk, 256, 4096), 256, 0, st>>>(A.items, n_blk, ik, ii);
            size_t sb = 0;
            CK(cub::DeviceRadixSort::SortPairs(nullptr, sb, ik, ik2, ii, ii2, n_blk, 0, 32, st));
            char* stmp; CKR(t2.get(&stmp, sb));
            CK(cub::DeviceRadixSort::SortPairs(stmp, sb, ik, ik2, ii, ii2, n_blk, 0, 32, st));
            k_item_gather<<<grid_for(n_blk, 256, 4096), 256, 0, st>>>(ii2, n_blk, A.items, A.items_x, A.item_blk);
        }
        // ---- norms, tables, w^
        CKR(dmalloc(P, &P->nD, (size_t)n_rows)); CKR(dmalloc(P, &P->nL, (size_t)n_rows)); CKR(dmalloc(P, &P->nT, (size_t)n_rows));
        CK(cudaMemsetAsync(P->nD, 0, (size_t)(n_rows ? n_rows : 1) * 8, st)); CK(cudaMemsetAsync(P->nL, 0, (size_t)(n_rows ? n_rows : 1) * 8, st));
        CK(cudaMemsetAsync(P->nT, 0, (size_t)(n_rows ? n_rows : 1) * 8, st));
        CKR(dmalloc(P, &P->mode_union, (size_t)ns)); CKR(dmalloc(P, &P->mode_con, (size_t)ns)); CKR(dmalloc(P, &P->mode_cost, (size_t)ns));
        CKR(dmalloc(P, &P->mode_fixed, (size_t)ns * 4));
        CKR(dmalloc(P, &P->st, 1));
        CK(cudaMemsetAsync(P->st, 0, sizeof(DevState), st));
        if (n_blk) {
            k_norms<<<grid_for(n_blk * 32, 256, 1 << 16), 256, 0, st>>>(n_blk, Rb, A.start, A.len, A.seg, A.valD, A.valL, P->tab, P->nD, P->nL, P->nT);
            k_count_sets<<<grid_for(n_rows, 256, 4096), 256, 0, st>>>(n_rows, A.rseg, rlen, P->nD, P->nL, P->nT, P->tab);
            k_count_entries<<<grid_for(n_blk, 256, 4096), 256, 0, st>>>(n_blk, A.seg, A.ulen, P->tab);
        }
        k_finish_tables<<<1, 1, 0, st>>>(P->tab, n_struct, P->st, P->mode_union, P->mode_con, P->mode_cost, P->mode_fixed, ns);
        state_init(P);
        CK(cudaMemcpyAsync(P->h_tab.data(), P->tab, sizeof(StructInfo) * ns, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        CK(cudaGetLastError());
    }
    // ---- vectors
    const long long NR = A.n_rows;
    CKR(dmalloc(P, &P->x, (size_t)S)); CKR(dmalloc(P, &P->g, (size_t)S + 8)); CKR(dmalloc(P, &P->xtmp, (size_t)S));
    CKR(dmalloc(P, &P->rbuf, (size_t)S + 8));
    CK(cudaMemsetAsync(P->rbuf, 0, ((size_t)S + 8) * 8, st));
    CKR(dmalloc(P, &P->xstage, (size_t)S));
    CK(cudaMemsetAsync(P->x, 0, (S ? S : 1) * 8, st)); CK(cudaMemsetAsync(P->g, 0, ((size_t)S + 8) * 8, st));
    double** vecs[] = {&P->d, &P->l, &P->Dg, &P->Lg};
    for (auto pp : vecs) { CKR(dmalloc(P, pp, (size_t)NR)); CK(cudaMemsetAsync(*pp, 0, (NR ? NR : 1) * 8, st)); }
    CKR(gv_alloc(P, &P->pq, (size_t)NR)); CKR(gv_alloc(P, &P->uv, (size_t)NR));
    const size_t npart = (size_t)(A.n > MAX_PARTIALS ? A.n : MAX_PARTIALS);     // per block row (forward epilogues) or per CTA
    CKR(dmalloc(P, &P->cpart, npart));
    CKR(dmalloc(P, &P->wq, 1));
    CK(cudaMemsetAsync(P->wq, 0, sizeof(WorkQueue), st));
    CKR(dmalloc(P, &P->live8, (size_t)(P->act.n ? P->act.n : 1)));
    CK(cudaMemsetAsync(P->live8, 1, (size_t)(P->act.n ? P->act.n : 1), st));      // until a residual pass has written it: every block row
    CKR(dmalloc(P, &P->live_count, 1));
    CK(cudaMemsetAsync(P->live_count, 0, sizeof(unsigned long long), st));
    CKR(dmalloc(P, &P->gpart, (size_t)(S / 256 + 2)));
    CK(cudaMemsetAsync(P->gpart, 0, (size_t)(S / 256 + 2) * 8, st)); CKR(dmalloc(P, &P->part_prox, npart));
    CKR(dmalloc(P, &P->part_phi, npart)); CKR(dmalloc(P, &P->part_cnt, npart));
    CKR(dmalloc(P, &P->sink, 4));
    CK(cudaMemsetAsync(P->cpart, 0, npart * 8, st));
    CK(cudaMemsetAsync(P->part_prox, 0, npart * 8, st)); CK(cudaMemsetAsync(P->part_phi, 0, npart * 8, st));
    CK(cudaMemsetAsync(P->part_cnt, 0, npart * 8, st));
    // ---- CSR of the transposes restricted to the labelled rows
    CKR(build_transpose(P, A));
    if (P->value_bits == 16) {              // half copies of the arrays the iteration streams (the fp32 ones stay for set-up work)
        const size_t na = (size_t)(A.entries_padded ? A.entries_padded : 4) * A.R, nt = (size_t)(A.t_entries_padded ? A.t_entries_padded : 4) * A.R;
        CKR(dmalloc(P, &A.valD16, na)); CKR(dmalloc(P, &A.valL16, na)); CKR(dmalloc(P, &A.t_valD16, nt)); CKR(dmalloc(P, &A.t_valL16, nt));
        k_to_half<<<P->sm_count * 8, 256, 0, st>>>(A.valD, A.valD16, na); k_to_half<<<P->sm_count * 8, 256, 0, st>>>(A.valL, A.valL16, na);
        k_to_half<<<P->sm_count * 8, 256, 0, st>>>(A.t_valD, A.t_valD16, nt); k_to_half<<<P->sm_count * 8, 256, 0, st>>>(A.t_valL, A.t_valL16, nt);
        CK(cudaGetLastError());
        int over = 0;
        CK(cudaMemcpyAsync(&over, flag + 2, sizeof(int), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        if (over) return FREDOPT_INVALID_ARG;                    // a value beyond the range of a half
    }
    compute_pass_bytes(P);
    CK(cudaStreamSynchronize(st));
    return FREDOPT_OK;
}

extern "C" {

int fredopt_shard_range(const int64_t* row_ptr, const int32_t* voxel_labels, int64_t n_rows, int32_t rank, int32_t world,
                        int64_t* v_begin, int64_t* v_end) {
    if (!row_ptr || (n_rows > 0 && !voxel_labels) || n_rows < 0 || world < 1 || rank < 0 || rank >= world || !v_begin || !v_end)
        return FREDOPT_INVALID_ARG;
    long long total = 0;
    for (int64_t i = 0; i < n_rows; ++i) if (voxel_labels[i] != 0) total += row_ptr[i + 1] - row_ptr[i] + 1;
    // cut r: the first voxel at which the running weight reaches ceil(r * total / world); cut 0 = 0, cut world = n_rows
    auto cut = [&](int r) -> int64_t {
        if (r <= 0) return 0;
        if (r >= world) return n_rows;
        const long long target = (long long)(((__int128)total * r + world - 1) / world);
        long long run = 0;
        for (int64_t i = 0; i < n_rows; ++i) {
            if (run >= target) return i;
            if (voxel_labels[i] != 0) run += row_ptr[i + 1] - row_ptr[i] + 1;
        }
        return n_rows;
    };
    *v_begin = cut(rank);
    *v_end = cut(rank + 1);
    return FREDOPT_OK;
}

int fredopt_set_reduce(fredopt_plan* P, fredopt_reduce_fn fn, void* ctx) {
    if (!P) return FREDOPT_INVALID_ARG;
    P->reduce_fn = fn; P->reduce_ctx = ctx;
    invalidate_graphs(P);
    if (!fn || P->shard_world <= 1) return FREDOPT_OK;
    return recount_sets(P, false);        // local counts, then (sharded) their sum over the ranks -> W, w^ of the whole plan
}

int fredopt_create(const fredopt_csr* D, const fredopt_csr* L, const int32_t* voxel_labels, const fredopt_bounds* bounds,
                   int32_t n_struct, void* cuda_stream, fredopt_plan** out) {
    return fredopt_create_ex(D, L, voxel_labels, bounds, n_struct, cuda_stream, nullptr, out);
}

int fredopt_create_ex(const fredopt_csr* D, const fredopt_csr* L, const int32_t* voxel_labels, const fredopt_bounds* bounds,
                      int32_t n_struct, void* cuda_stream, const fredopt_create_options* opt, fredopt_plan** out) {
    if (!out) return FREDOPT_INVALID_ARG;
    *out = nullptr;
    fredopt_create_options o;
    memset(&o, 0, sizeof(o));
    if (opt) {
        if (opt->struct_size < (int32_t)(2 * sizeof(int32_t)) || opt->struct_size > (int32_t)sizeof(o)) return FREDOPT_INVALID_ARG;
        memcpy(&o, opt, (size_t)opt->struct_size);
    }
    if (o.index_width != 0 && o.index_width != 32) return FREDOPT_INVALID_ARG;
    if (o.block_rows != 0 && o.block_rows != 1 && o.block_rows != 2 && o.block_rows != 4) return FREDOPT_INVALID_ARG;
    if (o.value_bits != 0 && o.value_bits != 32 && o.value_bits != 16) return FREDOPT_INVALID_ARG;
    if (o.shard_world < 0 || o.shard_rank < 0 || (o.shard_world == 0 && o.shard_rank != 0) || (o.shard_world > 0 && o.shard_rank >= o.shard_world))
        return FREDOPT_INVALID_ARG;
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
    P->force_idx32 = o.index_width == 32;
    P->block_rows_opt = o.block_rows;
    P->value_bits = o.value_bits == 16 ? 16 : 32;
    P->shard_rank = o.shard_rank; P->shard_world = o.shard_world > 1 ? o.shard_world : 1;
    int rc = create_impl(P, D, L, voxel_labels, bounds, n_struct);
    if (rc != FREDOPT_OK) { fredopt_destroy(P); return rc; }
    *out = P;
    return FREDOPT_OK;
}

}  // extern "C"
