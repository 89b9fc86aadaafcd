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

int build_transpose(fredopt_plan* P, RowSet& R) {
    cudaStream_t st = P->stream;
    const long long n = R.n, S = P->S;
    // 16-bit row indices: cut every (segment, spot) run where the row index crosses a multiple of 65536
    int H = (int)((n + 65535) >> 16);
    if (H < 1) H = 1;
    bool idx16 = R.n_seg < 256 && H < (1 << 23) && (double)S * R.n_seg * H < 4.0e9 && !P->force_idx32;
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


// ============================================================================================ API
extern "C" {

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
        if (S <= 65536 && !P->force_idx32) {   // 16-bit column indices for the hot kernels
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
        if (S <= 65536 && !P->force_idx32) {
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
    state_init(P);
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
    int rc = create_impl(P, D, L, voxel_labels, bounds, n_struct);
    if (rc != FREDOPT_OK) { fredopt_destroy(P); return rc; }
    *out = P;
    return FREDOPT_OK;
}

}  // extern "C"
