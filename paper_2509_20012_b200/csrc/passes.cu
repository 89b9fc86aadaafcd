// passes.cu -- the calls of include/fredopt.h outside the iteration: spot weights, fredopt_dose_let (Eq. 1), fredopt_proximity,
// the per-pass exports (per-SpMV parity, configs[4] sweep), the evaluation quantities (DVH / LVH / cDLVH, cDL30, Table 1) and
// the streaming-read ceiling.  Argument checking and staging of host buffers; every step runs in the kernels.
#include "fredopt_plan.cuh"
#include "kernels_eval.cuh"

#include <cub/cub.cuh>

thread_local std::string g_last_cuda_error;

#ifdef FREDOPT_CHECKED
void chk_upload_passes(const ChkRange* h, int n) { chk_upload_tu(h, n); }
#endif

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

int fredopt_set_weights_f64(fredopt_plan* P, const double* x) {
    if (!P || !x) return FREDOPT_INVALID_ARG;
    const bool dev = is_device_ptr(x);
    CK(cudaMemcpyAsync(P->x, x, P->S * 8, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, P->stream));
    if (!dev) CK(cudaStreamSynchronize(P->stream));       // the caller's array is borrowed for the call only
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

int fredopt_iterate_host(fredopt_plan* P, int32_t n_iter, float lambda, float beta0, float a, const float* x_in, float* x_out,
                         fredopt_stats* stats) {
    if (!P) return FREDOPT_INVALID_ARG;
    // everything is enqueued on the plan's stream; the caller's arrays are borrowed until the one synchronisation at the end
    bool pending_host_copy = false;
    if (x_in) {
        const float* dx = x_in;
        if (!is_device_ptr(x_in)) {
            CK(cudaMemcpyAsync(P->xstage, x_in, (size_t)P->S * 4, cudaMemcpyHostToDevice, P->stream));
            dx = P->xstage;
            pending_host_copy = true;
        }
        k_f32_to_f64<<<grid_for(P->S, 256, 1024), 256, 0, P->stream>>>(dx, P->x, P->S);
        ++P->launches;
    }
    const int rc = fredopt_iterate(P, n_iter, lambda, beta0, a);
    if (rc != FREDOPT_OK) {
        if (pending_host_copy) cudaStreamSynchronize(P->stream);
        return rc;
    }
    if (x_out) {
        if (is_device_ptr(x_out)) {
            k_f64_to_f32<<<grid_for(P->S, 256, 1024), 256, 0, P->stream>>>(P->x, x_out, P->S);
            ++P->launches;
        } else {
            float* tmp = (float*)P->xtmp;   // S doubles of scratch hold S floats
            k_f64_to_f32<<<grid_for(P->S, 256, 1024), 256, 0, P->stream>>>(P->x, tmp, P->S);
            ++P->launches;
            CK(cudaMemcpyAsync(x_out, tmp, (size_t)P->S * 4, cudaMemcpyDeviceToHost, P->stream));
        }
    }
    if (stats) {
        if (!P->st_host) CK(cudaMallocHost((void**)&P->st_host, sizeof(DevState)));
        CK(cudaMemcpyAsync(P->st_host, P->st, sizeof(DevState), cudaMemcpyDeviceToHost, P->stream));
    }
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(P->stream));
    if (stats) fill_stats(P, *P->st_host, stats);
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
    // d, l: caller outputs (host or device), voxel-indexed, n_rows floats; rows outside R are 0.  Host outputs are staged through a
    // buffer the plan owns (allocated at the first such call, kept)
    float *dd = d, *dl = l;
    const bool hd = d && !is_device_ptr(d), hl = l && !is_device_ptr(l);
    if ((hd || hl) && !P->out_stage) CKR(dmalloc(P, &P->out_stage, 2 * (size_t)(P->V ? P->V : 1)));
    chk_sync(P->stream);                 // checked build: the allocation table on the device is current
    if (hd) dd = P->out_stage;
    if (hl) dl = P->out_stage + (P->V ? P->V : 1);
    if (dd) cudaMemsetAsync(dd, 0, (size_t)P->V * 4, P->stream);
    if (dl) cudaMemsetAsync(dl, 0, (size_t)P->V * 4, P->stream);
    if (R.n) {
        const uint8_t* md = P->mode_fixed + (size_t)m * P->max_seg;
        const GatherVec none{nullptr, nullptr, nullptr};
        const bool i16 = R.col16 != nullptr;
        const void* colp = R.colp();
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
        launch_fwd_kernel(P, EPI_F32VOX, R, 0, n_long, md, xd, nullptr, nullptr, none, nullptr, nullptr, dd, dl, letd_out, NO_RESID);
    }
    int rc = FREDOPT_OK;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && hd) e = cudaMemcpyAsync(d, dd, (size_t)P->V * 4, cudaMemcpyDeviceToHost, P->stream);
    if (e == cudaSuccess && hl) e = cudaMemcpyAsync(l, dl, (size_t)P->V * 4, cudaMemcpyDeviceToHost, P->stream);
    if (hd || hl) { cudaError_t e2 = cudaStreamSynchronize(P->stream); if (e == cudaSuccess) e = e2; }
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
        if (!P->fullUV.pair) CKR(gv_alloc(P, &P->fullUV, (size_t)R.n_rows));
        chk_sync(P->stream);
        vec = P->fullUV;
    }
    const float *du = nullptr, *dv = nullptr; void *fu = nullptr, *fv = nullptr;
    if (u) CKR(stage_in_f32(P, u, P->V, &du, &fu));
    if (v) { int rc = stage_in_f32(P, v, P->V, &dv, &fv); if (rc) { cudaFree(fu); return rc; } }
    if (R.n_rows) { k_gather_uv<<<grid_for(R.n_rows, 256, 4096), 256, 0, P->stream>>>(du, dv, R.vox, vec, R.n_rows); ++P->launches; }
    float* dout = out; void* fo = nullptr;
    if (!is_device_ptr(out)) { cudaError_t e = cudaMalloc(&fo, (P->S ? P->S : 1) * 4); if (e != cudaSuccess) { cudaFree(fu); cudaFree(fv); CK(e); } dout = (float*)fo; }
    const int m = (u ? 1 : 0) | (v ? 2 : 0);
    cudaMemsetAsync(dout, 0, (size_t)(P->S ? P->S : 1) * 4, P->stream);     // spots without entries are never visited
    launch_transpose(P, TEPI_F32, R, P->mode_fixed + (size_t)m * P->max_seg, vec, nullptr, nullptr, dout);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && fo) e = cudaMemcpyAsync(out, dout, P->S * 4, cudaMemcpyDeviceToHost, P->stream);
    if (fo || fu || fv) { cudaError_t e2 = cudaStreamSynchronize(P->stream); if (e == cudaSuccess) e = e2; }
    cudaFree(fo); cudaFree(fu); cudaFree(fv);
    CK(e);
    return FREDOPT_OK;
}

int fredopt_set_voxel_bounds(fredopt_plan* P, int32_t field, const float* values) {
    if (!P || field < 0 || field >= VB_N) return FREDOPT_INVALID_ARG;
    const RowSet& A = P->act;
    cudaStream_t st = P->stream;
    VoxBounds nv = P->vb;
    double* nbuf = nullptr;
    if (values) {
        const float* dv; void* fr = nullptr;
        CKR(stage_in_f32(P, values, P->V, &dv, &fr));
        cudaError_t e = cudaMalloc((void**)&nbuf, (size_t)(A.n_rows ? A.n_rows : 1) * 8);
        int* bad = nullptr;
        if (e == cudaSuccess) e = cudaMalloc((void**)&bad, sizeof(int));
        int hbad = 0;
        if (e == cudaSuccess) e = cudaMemsetAsync(bad, 0, sizeof(int), st);
        if (e == cudaSuccess) {
            nv.f[field] = nbuf;
            if (A.n_rows) {
                k_vb_fill<<<grid_for(A.n_rows, 256, 4096), 256, 0, st>>>(A.n_rows, A.vox, A.rseg, P->tab, field, dv, nbuf, bad);
                k_vb_check<<<grid_for(A.n_rows, 256, 4096), 256, 0, st>>>(A.n_rows, A.rseg, P->tab, nv, bad);
                P->launches += 2;
            }
            e = cudaMemcpyAsync(&hbad, bad, sizeof(int), cudaMemcpyDeviceToHost, st);
        }
        cudaError_t e2 = cudaStreamSynchronize(st);
        if (e == cudaSuccess) e = e2;
        if (e == cudaSuccess) e = cudaGetLastError();
        cudaFree(bad); cudaFree(fr);
        if (e != cudaSuccess || hbad) { cudaFree(nbuf); if (e != cudaSuccess) CK(e); return FREDOPT_INVALID_ARG; }   // state untouched
    } else {
        nv.f[field] = nullptr;
    }
    CK(cudaStreamSynchronize(st));                        // nothing in flight reads the old array
    cudaFree(P->vb_buf[field]);
    P->vb_buf[field] = nbuf;
    P->vb = nv;
    invalidate_graphs(P);                                 // captured launches hold the old pointers
    if (field == VB_LETD_MAX) CKR(recount_sets(P, true)); // the LETd rows L_i - LETmax_i D_i changed: norms, participating sets, w^
    return FREDOPT_OK;
}

int fredopt_proximity(fredopt_plan* P, const float* x, double* prox, int64_t* n_violated) {
    if (!P || (!prox && !n_violated)) return FREDOPT_INVALID_ARG;
    const double* xd;
    CKR(resolve_x(P, x, &xd));
    // scratch: Dg / Lg hold the products so that the iteration's d, l are left alone
    launch_forward(P, P->act, P->mode_con, xd, P->Dg, P->Lg, EPI_RESID, 0);     // a11: one pass, statistics only
    if (P->shard_world > 1) {      // local statistics -> the caller's reduction
        if (!P->reduce_fn) return FREDOPT_INVALID_ARG;
        const int np = P->act.n ? (int)P->act.n : 0;
        launch_sum_to(P, P->rbuf, P->part_prox, nullptr, np);
        launch_sum_to(P, P->rbuf + 1, nullptr, P->part_cnt, np);
        CKR(reduce_call(P, P->rbuf, 2));
        double h2[2];
        CK(cudaMemcpyAsync(h2, P->rbuf, 16, cudaMemcpyDeviceToHost, P->stream));
        CK(cudaStreamSynchronize(P->stream));
        CK(cudaGetLastError());
        if (prox) *prox = h2[0];
        if (n_violated) *n_violated = (int64_t)h2[1];
        return FREDOPT_OK;
    }
    launch_finalize(P, P->act.n ? (int)P->act.n : 1);
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
    if (P->shard_world > 1) return FREDOPT_UNSUPPORTED;          // a structure's voxels are spread over the ranks
    const double* xd;
    CKR(resolve_x(P, x, &xd));
    const long long rb = P->row_base[label - 1];                 // the structure's real rows; padding rows follow them
    const long long nr = (long long)P->h_tab[label - 1].rows;
    *rb_out = rb; *nr_out = nr;
    if (nr == 0) return FREDOPT_OK;
    const RowSet& A = P->act;
    const int m = quantity == 0 ? 1 : quantity == 1 ? 2 : 3;
    const uint8_t* md = P->mode_fixed + (size_t)m * P->max_seg;
    const GatherVec none{nullptr, nullptr, nullptr};
    launch_fwd_kernel(P, EPI_STORE, A, rb / A.R, (nr + A.R - 1) / A.R, md, xd, P->Dg + rb, P->Lg + rb, none, nullptr, nullptr, nullptr, nullptr, 0,
                      NO_RESID);
    k_quantity<<<grid_for(nr, 256, 1024), 256, 0, P->stream>>>(nr, quantity, P->Dg + rb, P->Lg + rb, P->uv.cD + rb);
    ++P->launches;
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
