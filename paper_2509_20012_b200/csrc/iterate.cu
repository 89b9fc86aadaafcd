// iterate.cu -- launches of the hot kernels and the orchestration of fredopt_iterate: one iteration of SuperiorDLET (Fig. 3,
// PAPER.md:165-199) around the AMSrelaxDLET step (Fig. 2) as a replayed CUDA graph; options, statistics,
// per-pass timing.
#include "fredopt_plan.cuh"
#include "kernels_iter.cuh"

#include <nvtx3/nvToolsExt.h>

// ============================================================================================ launches
// Every pass is bracketed by an NVTX range (visible in a timeline tool; a few nanoseconds without one) and, with
// FREDOPT_OPT_TIME_PASSES, by a pair of CUDA events taken from a pool the plan keeps.
static const char* const PASS_LABEL[FREDOPT_N_PASSES] = {"fredopt F1 forward_x", "fredopt T1 transpose_g", "fredopt F2 forward_g",
                                                         "fredopt select", "fredopt residual", "fredopt T2 transpose_b"};
static void ev_begin(fredopt_plan* P, int pass) {
    nvtxRangePushA(PASS_LABEL[pass]);
    if (!P->time_passes) return;
    EventPair ep;
    if (!P->event_pool.empty()) { ep = P->event_pool.back(); P->event_pool.pop_back(); }
    else { cudaEventCreate(&ep.a); cudaEventCreate(&ep.b); }
    ep.pass = pass;
    cudaEventRecord(ep.a, P->stream);
    P->events.push_back(ep);
}
// values a back-projection over `items` needs with the liveness bytes `live` (added to *live_count)
static void launch_count_live(fredopt_plan* P, const Item* items, const uint8_t* mode, const uint8_t* live) {
    const RowSet& R = P->act;
    const void* tc = R.t_col16 ? (const void*)R.t_col16 : (const void*)R.t_col;
    const bool i16 = R.t_col16 != nullptr;
    const long long n = R.t_n_items;
#define CNT_CALL(RB, I16) k_count_live<RB, I16><<<P->sm_count * 8, FWD_THREADS, 0, P->stream>>>(n, items, mode, tc, live, P->live_count)
    switch (R.R) {
        case 1: if (i16) { CNT_CALL(1, true); } else { CNT_CALL(1, false); } break;
        case 2: if (i16) { CNT_CALL(2, true); } else { CNT_CALL(2, false); } break;
        default: if (i16) { CNT_CALL(4, true); } else { CNT_CALL(4, false); } break;
    }
#undef CNT_CALL
}
static void ev_end(fredopt_plan* P) {
    nvtxRangePop();
    if (!P->time_passes) return;
    cudaEventRecord(P->events.back().b, P->stream);
    if (P->count_pending) {                 // after the bracket: the count is not part of the timed pass
        P->count_pending = false;
        launch_count_live(P, P->count_items, P->count_mode, P->live8);
        ++P->live_launches;
    }
}

// grid of the item kernels: persistent, one CTA per resident slot (launch bounds of k_forward / k_transpose); the items come
// from the work queue
constexpr int GRAPH_UNROLL = 8;       // iterations captured into the long graph
int fwd_grid(fredopt_plan* P, long long n) {
    return grid_for(n, FWD_WARPS, P->sm_count * FWD_MIN_CTAS);
}
// static round-robin form of the item kernels (no queue): two waves of the resident CTAs
#ifndef STATIC_WAVES
#define STATIC_WAVES 2
#endif
static int static_grid(fredopt_plan* P, long long n) { return grid_for(n, FWD_WARPS, P->sm_count * FWD_MIN_CTAS * STATIC_WAVES); }


const ResidArgs NO_RESID{nullptr, nullptr, nullptr, GatherVec{nullptr, nullptr, nullptr}, nullptr, nullptr, nullptr, nullptr, nullptr};

// k_forward<EPI, R, I16> over n block rows of R starting at block row b0 (per-row arguments are passed already offset by the
// caller: oD, oL, vox point at row b0 * R)
#define FREDOPT_DISPATCH(RB, I16, CALL)                                             \
    switch (RB) {                                                                   \
        case 1: if (I16) { CALL(1, true); } else { CALL(1, false); } break;         \
        case 2: if (I16) { CALL(2, true); } else { CALL(2, false); } break;         \
        default: if (I16) { CALL(4, true); } else { CALL(4, false); } break;        \
    }
#ifdef FREDOPT_CHECKED
void chk_upload_iterate(const ChkRange* h, int n) { chk_upload_tu(h, n); }
#endif
void launch_fwd_kernel(fredopt_plan* P, int epi, const RowSet& R, long long b0, long long n, const uint8_t* mode, const double* x,
                       double* oD, double* oL, const GatherVec& pq, const StructInfo* tab, double* cpart, float* fD, float* fL,
                       int letd_out, const ResidArgs& ra) {
    if (n <= 0) return;
    chk_sync(P->stream);
    // Items from the queue or dealt statically: FREDOPT_OPT_WORK_QUEUE decides if it was set; otherwise the queue is used where it
    // pays -- enough items to balance (at least 6 per resident warp) and long ones (2 048 values on average): with short rows the
    // one counter every warp increments per item becomes the bottleneck (isolated forward pass over all rows, 2.9e8 non-zeros, mean
    // row 900: 2.5 TB/s from the queue, 5.1 TB/s dealt statically), with few items there is nothing to balance.
    const bool dyn = P->fwd_dynamic >= 0 ? P->fwd_dynamic != 0
                                         : (R.n >= 6LL * P->sm_count * FWD_MIN_CTAS * FWD_WARPS && R.entries_padded * R.R >= 2048LL * R.n);
    WorkQueue* wq = dyn ? P->wq : nullptr;
    const int g = wq ? fwd_grid(P, n) : static_grid(P, n);
    const bool whole = P->fwd_sorted && b0 == 0 && n == R.n && R.items_x;   // whole set: longest-first execution order
    const Item* items = whole ? R.items_x : R.items + b0;
    const int32_t* iblk = whole ? R.item_blk : nullptr;
    const int32_t* vox = R.vox ? R.vox + b0 * R.R : nullptr;
    const void* col = R.colp();
    const bool i16 = R.col16 != nullptr;
#define FWD_ARGS(VD, VL) g, FWD_THREADS, n, items, iblk, wq, vox, mode, col, VD, VL, x, oD, oL, pq, tab, P->vb, cpart, P->st, fD, fL, letd_out, ra
#define FWD_CALL_VT(RB, I16, VT, VD, VL)                                                          \
    switch (epi) {                                                                                \
        case EPI_STORE: klaunch(P, k_forward<EPI_STORE, RB, I16, VT>, FWD_ARGS(VD, VL)); break;    \
        case EPI_STORE_PQ: klaunch(P, k_forward<EPI_STORE_PQ, RB, I16, VT>, FWD_ARGS(VD, VL)); break; \
        case EPI_CPART: klaunch(P, k_forward<EPI_CPART, RB, I16, VT>, FWD_ARGS(VD, VL)); break;    \
        case EPI_F32VOX: klaunch(P, k_forward<EPI_F32VOX, RB, I16, VT>, FWD_ARGS(VD, VL)); break;  \
        default: klaunch(P, k_forward<EPI_RESID, RB, I16, VT>, FWD_ARGS(VD, VL)); break;           \
    }
#define FWD_CALL(RB, I16)                                                                         \
    if (R.valD16) { FWD_CALL_VT(RB, I16, __half, (const __half*)R.valD16, (const __half*)R.valL16) } \
    else { FWD_CALL_VT(RB, I16, float, (const float*)R.valD, (const float*)R.valL) }
    FREDOPT_DISPATCH(R.R, i16, FWD_CALL)
#undef FWD_CALL_VT
#undef FWD_ARGS
#undef FWD_CALL
}

// k_transpose<R, I16> over n work items
void launch_tr_kernel(fredopt_plan* P, const RowSet& R, const Item* items, const int32_t* slots, long long n, const uint8_t* mode,
                      const GatherVec& vec, const uint8_t* live) {
    if (n <= 0) return;
    chk_sync(P->stream);
    WorkQueue* wq = P->tr_dynamic ? P->wq : nullptr;
    const int g = wq ? fwd_grid(P, n) : static_grid(P, n);
    const void* tc = R.t_col16 ? (const void*)R.t_col16 : (const void*)R.t_col;
    const bool i16 = R.t_col16 != nullptr;
    if (!P->skip_dead) live = nullptr;
#define TR_CALL_VT(RB, I16, VT, TD, TL)                                                                                         \
    if (live) klaunch(P, k_transpose<RB, I16, true, VT>, g, FWD_THREADS, n, items, slots, wq, mode, tc, TD, TL, vec, R.t_partial, live); \
    else klaunch(P, k_transpose<RB, I16, false, VT>, g, FWD_THREADS, n, items, slots, wq, mode, tc, TD, TL, vec, R.t_partial, live);
#define TR_CALL(RB, I16)                                                                                                         \
    if (R.t_valD16) { TR_CALL_VT(RB, I16, __half, (const __half*)R.t_valD16, (const __half*)R.t_valL16) }                        \
    else { TR_CALL_VT(RB, I16, float, (const float*)R.t_valD, (const float*)R.t_valL) }
    FREDOPT_DISPATCH(R.R, i16, TR_CALL)
#undef TR_CALL_VT
#undef TR_CALL
    if (live && P->time_passes && P->live_count && &R == &P->act && n == R.t_n_items) {
        // measurement: what this launch needed, counted by a separate kernel; launch_transpose closes the timed bracket first
        P->count_pending = true; P->count_items = items; P->count_mode = mode;
    }
}

// epi: EPI_STORE (d, l), EPI_STORE_PQ (d, l, the cost residuals p, q and partial sums of chi^2), EPI_CPART (Dg, Lg and partial
// sums of c), EPI_RESID (d, l and the residual / violation epilogue: step coefficients u, v if write_uv, statistics partials)
void launch_forward(fredopt_plan* P, const RowSet& R, const uint8_t* mode, const double* x, double* oD, double* oL, int epi,
                    int write_uv) {
    if (R.n == 0) {
        if (epi == EPI_CPART) cudaMemsetAsync(P->cpart, 0, 8, P->stream);
        if (epi == EPI_RESID) {   // nothing to visit: zero statistics (finalize reads one partial)
            cudaMemsetAsync(P->part_prox, 0, 8, P->stream); cudaMemsetAsync(P->part_phi, 0, 8, P->stream); cudaMemsetAsync(P->part_cnt, 0, 8, P->stream);
            if (write_uv) klaunch(P, k_sweep_end, grid_for(P->S, 256, 1 << 30), 256, P->S, P->x, P->st);   // k, eta^k still advance
        }
        return;
    }
    const GatherVec none{nullptr, nullptr, nullptr};
    ResidArgs ra = NO_RESID;
    if (epi == EPI_RESID) ra = ResidArgs{P->nD, P->nL, P->nT, write_uv ? P->uv : none, P->part_prox, P->part_phi, P->part_cnt, P->st, P->live8};
    launch_fwd_kernel(P, epi, R, 0, R.n, mode, x, oD, oL, epi == EPI_STORE_PQ ? P->pq : none, epi == EPI_STORE ? nullptr : P->tab,
                      epi == EPI_CPART ? P->cpart : epi == EPI_STORE_PQ ? P->part_phi : nullptr, nullptr, nullptr, 0, ra);
}
static int cpart_count(fredopt_plan* P) { return P->act.n ? (int)P->act.n : 1; }     // partial sums per block row

void launch_transpose(fredopt_plan* P, int tepi, const RowSet& R, const uint8_t* mode, const GatherVec& vec, double* g_out, double* x,
                      float* f_out, const uint8_t* live) {
    if (R.t_n_items == 0 && tepi != TEPI_UPDATE) return;          // nothing to add; the update still clamps (R6)
    if (P->tr_sorted) launch_tr_kernel(P, R, R.t_items, R.t_item_slot, R.t_n_items, mode, vec, live);
    else launch_tr_kernel(P, R, R.t_items_run, R.t_slot_run, R.t_n_items, mode, vec, live);
    const int gc = grid_for(P->S, 256, 1 << 30);
    if (tepi == TEPI_GRAD) klaunch(P, k_combine<TEPI_GRAD>, gc, 256, P->S, R.t_item_ptr, R.t_partial, g_out, P->gpart, x, P->st, f_out);
    else if (tepi == TEPI_UPDATE) klaunch(P, k_combine<TEPI_UPDATE>, gc, 256, P->S, R.t_item_ptr, R.t_partial, g_out, P->gpart, x, P->st, f_out);
    else klaunch(P, k_combine<TEPI_F32>, gc, 256, P->S, R.t_item_ptr, R.t_partial, g_out, P->gpart, x, P->st, f_out);
}

static int res_grid(fredopt_plan* P) {
    const int cap = P->sm_count * 4 < MAX_PARTIALS ? P->sm_count * 4 : MAX_PARTIALS;
    const long long n = P->act.n_rows > P->S ? P->act.n_rows : P->S;
    return grid_for(n, ROW_THREADS, cap);
}

static void launch_residual(fredopt_plan* P, double* d, double* l, int use_beta, int final, int write_uv) {
    const int g = res_grid(P);
    klaunch(P, k_residual, g, ROW_THREADS, P->act.n_rows, P->act.rseg, P->tab, P->vb, P->st, d, l, P->Dg, P->Lg, P->nD, P->nL, P->nT, P->uv, P->pq,
            P->x, P->g, P->S, P->part_prox, P->part_phi, P->part_cnt, use_beta, final, write_uv, P->live8, P->act.R);
}

// n_part: how many per-CTA partial sums the last residual pass wrote (k_residual: res_grid; forward epilogue: fwd_grid)
void launch_finalize(fredopt_plan* P, int n_part) {
    klaunch(P, k_finalize_stats, 1, 1024, P->st, P->part_prox, P->part_phi, P->part_cnt, n_part);
}

// Block-sequential AMS sweep (reading R23): Fig. 2's loop nest -- dose kind over the structures, then cDLET, then the LETd
// rows -- one (forward over the block's rows, residual, transposed over the block's items, update) group per block.
static void enqueue_block_sweep(fredopt_plan* P) {
    const RowSet& A = P->act;
    klaunch(P, k_sweep_begin, 1, 1, P->st);
    const int kind_flag[3] = {F_DOSE_SLAB, F_DL_SLAB, F_LETD};
    const int kind_mode[3] = {1, 2, 3};
    const GatherVec none{nullptr, nullptr, nullptr};
    for (int kind = 0; kind < 3; ++kind)
        for (int s = 0; s < P->n_struct; ++s) {
            const StructInfo& T = P->h_tab[s];
            if (!(T.flags & kind_flag[kind])) continue;
            const long long rb = P->row_base[s], nr = (long long)T.rows, re = rb + nr;     // real rows: padding rows follow them
            if (nr == 0) continue;
            const int RB = A.R;
            const uint8_t* md = P->mode_fixed + (size_t)kind_mode[kind] * P->max_seg;
            ev_begin(P, FREDOPT_PASS_FORWARD_X);
            launch_fwd_kernel(P, EPI_STORE, A, rb / RB, (nr + RB - 1) / RB, md, P->x, P->d + rb, P->l + rb, none, nullptr, nullptr, nullptr, nullptr, 0,
                              NO_RESID);
            ev_end(P);
            ev_begin(P, FREDOPT_PASS_RESIDUAL);
            const int gr = grid_for(nr, ROW_THREADS, P->sm_count * 4 < MAX_PARTIALS ? P->sm_count * 4 : MAX_PARTIALS);
            klaunch(P, k_block_residual, gr, ROW_THREADS, rb, re, s, kind, P->tab, P->vb, P->st, P->d, P->l, P->nD, P->nL, P->nT, P->uv, P->part_prox);
            ev_end(P);
            const long long m = (long long)T.part_kind[kind];
            const long long ib = A.t_seg_item_begin.empty() ? 0 : A.t_seg_item_begin[s], ie = A.t_seg_item_begin.empty() ? 0 : A.t_seg_item_begin[s + 1];
            if (m == 0) continue;                      // no row of the block has a non-zero norm: violations counted, no step
            ev_begin(P, FREDOPT_PASS_TRANSPOSE_B);
            launch_tr_kernel(P, A, A.t_items_seg + ib, A.t_slot_seg + ib, ie - ib, md, P->uv);
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
            launch_transpose(P, TEPI_GRAD, P->act, P->mode_cost, P->pq, P->g, nullptr, nullptr);       // a3: g = D^T p + L^T q
            ev_end(P);
            ev_begin(P, FREDOPT_PASS_FORWARD_G);
            launch_forward(P, P->act, P->mode_union, P->g, P->Dg, P->Lg, EPI_CPART);                   // a5: Dg, Lg, c
            ev_end(P);
            ev_begin(P, FREDOPT_PASS_SELECT);
            klaunch(P, k_select, 1, 1024, P->st, P->gpart, P->act.t_n_items ? grid_for(P->S, 256, 1 << 30) : 0, P->cpart, cpart_count(P),
                    P->part_phi, P->act.n == 0 ? 0 : t == 0 ? (int)P->act.n : res_grid(P), P->act.n_rows,
                    P->act.rseg, P->tab, P->vb, P->d, P->l, P->Dg, P->Lg);                                     // a4, a6: beta
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
    launch_transpose(P, TEPI_UPDATE, P->act, P->mode_con, P->uv, nullptr, P->x, nullptr, P->live8);    // a8, a9 (rows with a coefficient only)
    ev_end(P);
    return (int)(P->launches - before);
}


void launch_sum_to(fredopt_plan* P, double* out, const double* in, const long long* in_ll, int n) {
    if (in_ll) klaunch(P, k_sum_to_ll, 1, 1024, out, in_ll, n);
    else klaunch(P, k_sum_to, 1, 1024, out, in, n);
}

int reduce_call(fredopt_plan* P, double* buf, long long n) {
    if (!P->reduce_fn) return FREDOPT_INVALID_ARG;
    return P->reduce_fn(P->reduce_ctx, buf, (int64_t)n, (void*)P->stream) == 0 ? FREDOPT_OK : FREDOPT_CUDA_ERROR;
}

// One iteration of a SHARDED plan (simultaneous form): the local passes of enqueue_iteration with the sums over voxels completed
// by the caller's reduction -- the partial gradient (+ chi^2), c, and the partial step (+ statistics).  Launched directly.
static int enqueue_iteration_sharded(fredopt_plan* P, bool sa) {
    const RowSet& A = P->act;
    const long long S = P->S;
    const int gS = grid_for(S, 256, 1 << 30);
    if (sa) {
        launch_forward(P, A, P->mode_union, P->x, P->d, P->l, EPI_STORE_PQ);
        for (long long t = 0; t < P->reductionsN; ++t) {
            // local partial gradient into g (slots of the local rows), chi^2 of the local rows into g[S]
            if (A.t_n_items) launch_tr_kernel(P, A, A.t_items, A.t_item_slot, A.t_n_items, P->mode_cost, P->pq);
            klaunch(P, k_slots_sum, gS, 256, S, A.t_item_ptr, A.t_partial, P->g);
            klaunch(P, k_sum_to, 1, 1024, P->g + S, P->part_phi, A.n == 0 ? 0 : t == 0 ? (int)A.n : res_grid(P));
            CKR(reduce_call(P, P->g, S + 1));
            klaunch(P, k_gnorm, gS, 256, S, P->g, P->gpart);
            launch_forward(P, A, P->mode_union, P->g, P->Dg, P->Lg, EPI_CPART);
            klaunch(P, k_sum_to, 1, 1024, P->rbuf, P->cpart, A.n ? (int)A.n : 0);
            CKR(reduce_call(P, P->rbuf, 1));
            klaunch(P, k_select, 1, 1024, P->st, P->gpart, gS, P->rbuf, 1, P->g + S, 1, A.n_rows, A.rseg, P->tab, P->vb, P->d, P->l, P->Dg, P->Lg);
            const int last = t == P->reductionsN - 1;
            launch_residual(P, P->d, P->l, 1, last, last);
        }
    } else {
        launch_forward(P, A, P->mode_con, P->x, P->d, P->l, EPI_RESID, 1);
    }
    // local partial step and statistics -> reduction -> update + clamp on every rank
    if (A.t_n_items) launch_tr_kernel(P, A, A.t_items, A.t_item_slot, A.t_n_items, P->mode_con, P->uv, P->live8);
    klaunch(P, k_slots_sum, gS, 256, S, A.t_item_ptr, A.t_partial, P->rbuf);
    const int np = A.n == 0 ? 0 : sa ? res_grid(P) : (int)A.n;
    klaunch(P, k_sum_to, 1, 1024, P->rbuf + S, P->part_prox, np);
    klaunch(P, k_sum_to, 1, 1024, P->rbuf + S + 1, P->part_phi, np);
    klaunch(P, k_sum_to_ll, 1, 1024, P->rbuf + S + 2, P->part_cnt, np);
    CKR(reduce_call(P, P->rbuf, S + 3));
    klaunch(P, k_update_from, gS, 256, S, P->rbuf, P->x, P->st);
    return FREDOPT_OK;
}

void invalidate_graphs(fredopt_plan* P) {
    for (int i = 0; i < 8; ++i) if (P->gexec[i]) { cudaGraphExecDestroy(P->gexec[i]); P->gexec[i] = nullptr; }
}

void state_init(fredopt_plan* P) {
    k_set_params<<<1, 1, 0, P->stream>>>(P->st, 1.0, 0.0, 0.5, 1.0, 200, 1, 0, 2);
}

// ============================================================================================ API
void fill_stats(fredopt_plan* P, const DevState& h, fredopt_stats* out) {
    out->k = h.k; out->s = h.s; out->trials = h.trials; out->n_violated = h.n_viol;
    out->n_sets = h.n_sets; out->n_zero_norm_sets = h.n_zero;
    out->n_active_rows = P->act.n_true; out->nnz = P->nnz; out->nnz_active = P->act.nnz;
    out->block_rows = P->act.R; out->entries_active = P->act.entries;
    long long b = 0;
    const int sa_passes[] = {FREDOPT_PASS_FORWARD_X, FREDOPT_PASS_TRANSPOSE_G, FREDOPT_PASS_FORWARD_G, FREDOPT_PASS_SELECT,
                             FREDOPT_PASS_RESIDUAL, FREDOPT_PASS_TRANSPOSE_B};
    for (int p : sa_passes) b += P->pass_bytes[p];
    out->alg_bytes_iter = b;
    out->last_beta = h.last_beta; out->phi = h.phi; out->prox = h.prox; out->weight_sum = h.W;
}

extern "C" {

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
        case FREDOPT_OPT_WORK_QUEUE: {
            const int v = (int)value;
            if (v < 0 || v > 15) return FREDOPT_INVALID_ARG;
            P->fwd_dynamic = v & 1; P->tr_dynamic = (v >> 1) & 1; P->fwd_sorted = (v >> 2) & 1; P->tr_sorted = (v >> 3) & 1;
            for (int i = 0; i < 8; ++i) if (P->gexec[i]) { cudaGraphExecDestroy(P->gexec[i]); P->gexec[i] = nullptr; }
            break;
        }
        case FREDOPT_OPT_USE_PDL:
            if (P->use_pdl != (value != 0.0)) {            // the launch attribute is part of a captured graph: capture again
                P->use_pdl = value != 0.0;
                for (int i = 0; i < 8; ++i) if (P->gexec[i]) { cudaGraphExecDestroy(P->gexec[i]); P->gexec[i] = nullptr; }
            }
            break;
        case FREDOPT_OPT_BLOCK_SEQUENTIAL: P->block_sequential = value != 0.0; break;
        case FREDOPT_OPT_NORMALIZE_GRAD: P->normalize_grad = value != 0.0; break;
        case FREDOPT_OPT_ONE_SIDED_COST: P->one_sided_cost = value != 0.0; break;
        case FREDOPT_OPT_SKIP_SATISFIED:
            if (P->skip_dead != (value != 0.0)) {              // another kernel instantiation: capture again
                P->skip_dead = value != 0.0;
                invalidate_graphs(P);
            }
            break;
        case FREDOPT_OPT_TIME_PASSES:
            P->time_passes = value != 0.0;
            if (P->time_passes) {
                for (auto& ep : P->events) P->event_pool.push_back(ep);
                P->events.clear();
                for (int i = 0; i < FREDOPT_N_PASSES; ++i) { P->pass_ms[i] = 0; P->pass_launches[i] = 0; }
                P->live_launches = 0;
                if (P->live_count) cudaMemsetAsync(P->live_count, 0, sizeof(unsigned long long), P->stream);
            }
            break;
        default: return FREDOPT_INVALID_ARG;
    }
    return FREDOPT_OK;
}

int fredopt_iterate(fredopt_plan* P, int32_t n_iter, float lambda, float beta0, float a) {
    if (!P || n_iter < 0) return FREDOPT_INVALID_ARG;
    chk_sync(P->stream);                 // checked build: before any capture begins
    if (!(lambda > 0.f) || !(lambda <= 2.f) || !(beta0 >= 0.f) || !std::isfinite(beta0) || !(a > 0.f) || !(a < 1.f))
        return FREDOPT_INVALID_ARG;
    if (P->shard_world > 1 && !P->reduce_fn) return FREDOPT_INVALID_ARG;
    if (P->shard_world > 1 && P->block_sequential) return FREDOPT_UNSUPPORTED;
    // the step-size sequence beta0 a^s belongs to the plan (R8): the first superiorized call latches (beta0, a); calls with
    // beta0 = 0 neither latch nor consume it; a different pair needs FREDOPT_OPT_RESET
    int latch = 0;
    if (beta0 != 0.f && n_iter > 0) {
        if (!P->started) { latch = 1; P->latched_beta0 = beta0; P->latched_a = a; P->started = true; }
        else if (beta0 != P->latched_beta0 || a != P->latched_a) return FREDOPT_INVALID_ARG;
    }
    k_set_params<<<1, 1, 0, P->stream>>>(P->st, (double)lambda, (double)beta0, (double)a, P->eta, P->max_trials, P->accept_check,
                                           (P->normalize_grad ? SF_NORMALIZE_GRAD : 0) | (P->one_sided_cost ? SF_ONE_SIDED : 0), latch);
    ++P->launches;
    const bool sa = beta0 != 0.f;
    if (P->shard_world > 1) {                                   // one plan on several GPUs: direct launches + the caller's reduction
        if (n_iter > 0) {
            P->launch_err = cudaSuccess;
            for (int it = 0; it < n_iter; ++it) CKR(enqueue_iteration_sharded(P, sa));
            CK(P->launch_err);
        }
        CK(cudaGetLastError());
        return FREDOPT_OK;
    }
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
                    P->launch_err = cudaSuccess;
                    for (int r = 0; r < per; ++r) nk += enqueue_iteration(P, sa);
                    P->launches = l0;
                    cudaError_t e = cudaStreamEndCapture(P->stream, &gr);      // always ends the capture, also after a failed launch
                    if (e == cudaSuccess && P->launch_err != cudaSuccess) e = P->launch_err;
                    if (e != cudaSuccess) {                                    // nothing was enqueued: the plan's x, k, s are untouched
                        if (gr) cudaGraphDestroy(gr);
                        if (latch) P->started = false;
                        CK(e);
                    }
                    e = cudaGraphInstantiate(&P->gexec[gi], gr, 0);
                    cudaGraphDestroy(gr);
                    if (e != cudaSuccess) { P->gexec[gi] = nullptr; if (latch) P->started = false; }
                    CK(e);
                    P->gexec_red[gi] = P->reductionsN;
                    P->gexec_kernels[gi] = nk;
                }
                for (; left >= per; left -= per) { CK(cudaGraphLaunch(P->gexec[gi], P->stream)); P->launches += P->gexec_kernels[gi]; }
            }
        } else {
            P->launch_err = cudaSuccess;
            for (int it = 0; it < n_iter && P->launch_err == cudaSuccess; ++it) enqueue_iteration(P, sa);
            CK(P->launch_err);
        }
        if (!P->block_sequential)                         // block mode keeps its sweep statistics in the state already
            launch_finalize(P, sa ? res_grid(P) : (P->act.n ? (int)P->act.n : 1));
    }
    CK(cudaGetLastError());
    return FREDOPT_OK;
}

int fredopt_get_state(fredopt_plan* P, fredopt_state* out) {
    if (!P || !out) return FREDOPT_INVALID_ARG;
    DevState h;
    CK(cudaMemcpyAsync(&h, P->st, sizeof(DevState), cudaMemcpyDeviceToHost, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    out->k = h.k; out->s = h.s; out->trials = h.trials;
    out->beta_next = h.beta_next; out->eta_pow = h.eta_pow; out->last_beta = h.last_beta;
    out->beta0 = P->started ? P->latched_beta0 : 0.f; out->a = P->started ? P->latched_a : 0.f;
    out->latched = P->started ? 1 : 0;
    out->reserved = 0;
    return FREDOPT_OK;
}

int fredopt_set_state(fredopt_plan* P, const fredopt_state* in) {
    if (!P || !in) return FREDOPT_INVALID_ARG;
    if (in->k < 0 || in->s < 0 || in->trials < 0 || !(in->eta_pow >= 0.0) || !std::isfinite(in->eta_pow) || !(in->beta_next >= 0.0) ||
        !std::isfinite(in->beta_next) || !(in->last_beta >= 0.0) || !std::isfinite(in->last_beta) || (in->latched != 0 && in->latched != 1))
        return FREDOPT_INVALID_ARG;
    if (in->latched && (!(in->beta0 > 0.f) || !std::isfinite(in->beta0) || !(in->a > 0.f) || !(in->a < 1.f))) return FREDOPT_INVALID_ARG;
    DevState h;
    CK(cudaMemcpyAsync(&h, P->st, sizeof(DevState), cudaMemcpyDeviceToHost, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    h.k = in->k; h.s = in->s; h.trials = in->trials;
    h.beta_next = in->beta_next; h.eta_pow = in->eta_pow; h.last_beta = in->last_beta;
    if (in->latched) { h.beta0 = (double)in->beta0; h.a = (double)in->a; }
    CK(cudaMemcpyAsync(P->st, &h, sizeof(DevState), cudaMemcpyHostToDevice, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    P->started = in->latched != 0;
    P->latched_beta0 = in->latched ? in->beta0 : 0.f;
    P->latched_a = in->latched ? in->a : 0.f;
    return FREDOPT_OK;
}

int fredopt_get_stats(fredopt_plan* P, fredopt_stats* out) {
    if (!P || !out) return FREDOPT_INVALID_ARG;
    if (!P->st_host) CK(cudaMallocHost((void**)&P->st_host, sizeof(DevState)));
    CK(cudaMemcpyAsync(P->st_host, P->st, sizeof(DevState), cudaMemcpyDeviceToHost, P->stream));
    CK(cudaStreamSynchronize(P->stream));
    fill_stats(P, *P->st_host, out);
    return FREDOPT_OK;
}

int fredopt_get_pass_times(fredopt_plan* P, double* ms, int64_t* launches) {
    if (!P || !ms || !launches) return FREDOPT_INVALID_ARG;
    CK(cudaStreamSynchronize(P->stream));
    for (auto& ep : P->events) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, ep.a, ep.b) == cudaSuccess) { P->pass_ms[ep.pass] += t; P->pass_launches[ep.pass] += 1; }
        P->event_pool.push_back(ep);
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

int fredopt_get_pass_bytes_timed(fredopt_plan* P, int64_t* bytes) {
    if (!P || !bytes) return FREDOPT_INVALID_ARG;
    for (int i = 0; i < FREDOPT_N_PASSES; ++i) bytes[i] = P->pass_bytes[i];
    CK(cudaStreamSynchronize(P->stream));
    if (P->live_launches > 0 && P->act.t_n_items > 0) {
        unsigned long long cnt = 0;
        CK(cudaMemcpy(&cnt, P->live_count, sizeof(cnt), cudaMemcpyDeviceToHost));
        if (P->live_all < 0) {              // the same count with every block row live
            uint8_t* ones = nullptr;
            CK(cudaMalloc((void**)&ones, (size_t)(P->act.n ? P->act.n : 1)));
            cudaMemsetAsync(ones, 1, (size_t)(P->act.n ? P->act.n : 1), P->stream);
            cudaMemsetAsync(P->live_count, 0, sizeof(unsigned long long), P->stream);
            launch_count_live(P, P->tr_sorted ? P->act.t_items : P->act.t_items_run, P->mode_con, ones);
            unsigned long long all = 0;
            cudaMemcpyAsync(&all, P->live_count, sizeof(all), cudaMemcpyDeviceToHost, P->stream);
            cudaMemcpyAsync(P->live_count, &cnt, sizeof(cnt), cudaMemcpyHostToDevice, P->stream);   // put the running sum back
            CK(cudaStreamSynchronize(P->stream));
            cudaFree(ones);
            P->live_all = (long long)all;
        }
        if (P->live_all > 0) {
            const double frac = (double)cnt / ((double)P->live_launches * (double)P->live_all);
            bytes[FREDOPT_PASS_TRANSPOSE_B] = P->pass_bytes[FREDOPT_PASS_TRANSPOSE_B] - P->tr_con_value_bytes +
                                               (long long)(frac * (double)P->tr_con_value_bytes);
        }
    }
    return FREDOPT_OK;
}

int64_t fredopt_launch_count(fredopt_plan* P) { return P ? P->launches : 0; }


}  // extern "C"
