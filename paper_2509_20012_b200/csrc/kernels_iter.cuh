// kernels_iter.cuh -- the vector / scalar kernels of one iteration (launched from iterate.cu only): parameter latch, the
// accept loop of Fig. 3 on device scalars, the residual / violation pass of Fig. 2, the block-sequential form, statistics.
#pragma once
#include "fredopt_kernels.cuh"

namespace fredopt {

// ------------------------------------------------------------------------------------------ scalar kernels
__global__ void k_set_params(DevState* st, double lambda, double beta0, double a, double eta, long long max_trials,
                             int accept_check, int flags, int latch) {
    st->flags = flags;
    st->lambda = lambda;
    st->eta = eta;
    st->max_trials = max_trials;
    st->accept_check = accept_check;
    if (latch == 1) { st->beta0 = beta0; st->a = a; st->beta_next = beta0; }     // first superiorized call: beta_0 = beta0 (R8)
    if (latch == 2) { st->beta0 = 0.0; st->a = a; st->beta_next = 0.0; st->eta_pow = 1.0; }   // creation: eta^0 = 1
}

// chi^2 of Eq. (2) at x - b g from the stored products: d - b Dg, l - b Lg (exact: the products are linear in x).  All
// threads of the CTA take part; the value is valid in thread 0.
__device__ __forceinline__ double cost_along(double b, long long n, const int16_t* __restrict__ rseg,
                                             const StructInfo* __restrict__ tab, const VoxBounds& vb, const double* __restrict__ d,
                                             const double* __restrict__ l, const double* __restrict__ Dg,
                                             const double* __restrict__ Lg, int one_sided, double* sm) {
    double phi = 0.0;
    for (long long a = threadIdx.x; a < n; a += blockDim.x) {
        const int sg = rseg[a];
        if (sg < 0) continue;                                          // padding row of a ragged block
        const StructInfo& T = tab[sg];
        const double dref = vb.f[VB_DOSE_REF] ? vb.f[VB_DOSE_REF][a] : T.dose_ref;
        const double lref = vb.f[VB_DL_REF] ? vb.f[VB_DL_REF][a] : T.dl_ref;
        if (T.flags & F_DOSE_REF) { const double e = dref - fma(-b, Dg[a], d[a]); phi += T.what * e * e; }
        if (T.flags & F_DL_REF) { const double e = lref - fma(-b, Lg[a], l[a]); if (!(one_sided && e > 0.0)) phi += T.what * e * e; }
    }
    return block_sum(phi, sm);
}

// A thread's share of a fixed-order sum of n partial sums: elements t, t + T, t + 2T, ... (T threads), eight loads in flight
// at a time, added in index order.
__device__ __forceinline__ double strided_sum(const double* __restrict__ v, int n) {
    double acc = 0.0;
    const int T = blockDim.x;
    int i = threadIdx.x;
    for (; i + 7 * T < n; i += 8 * T) {
        double t[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) t[u] = v[i + u * T];
#pragma unroll
        for (int u = 0; u < 8; ++u) acc += t[u];
    }
    for (; i < n; i += T) acc += v[i];
    return acc;
}

// ---- sharded plans: local sums that go through the caller's reduction
// out[0] = fixed-order sum of in[0..n)   (one CTA)
__global__ void __launch_bounds__(1024) k_sum_to(double* __restrict__ out, const double* __restrict__ in, int n) {
    pdl_wait();
    pdl_trigger();
    __shared__ double sm[32];
    const double t = block_sum(strided_sum(in, n), sm);
    if (threadIdx.x == 0) out[0] = t;
}
__global__ void __launch_bounds__(1024) k_sum_to_ll(double* __restrict__ out, const long long* __restrict__ in, int n) {
    pdl_wait();
    pdl_trigger();
    __shared__ long long smc[32];
    long long c = 0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) c += in[i];
    const long long t = block_sum_ll(c, smc);
    if (threadIdx.x == 0) out[0] = (double)t;
}
// per-CTA partial sums of |g|^2 from the (reduced) gradient, in the layout k_select reads
__global__ void __launch_bounds__(256) k_gnorm(long long S, const double* __restrict__ g, double* __restrict__ gpart) {
    pdl_wait();
    pdl_trigger();
    __shared__ double sm[8];
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const double v = j < S ? g[j] : 0.0;
    const double q = block_sum(v * v, sm);
    if (threadIdx.x == 0) gpart[blockIdx.x] = q;
}
// out[j] = sum of the local partial-sum slots of spot j (0 for a spot without slots)
__global__ void __launch_bounds__(256) k_slots_sum(long long S, const long long* __restrict__ item_ptr, const double* __restrict__ partial,
                                                   double* __restrict__ out) {
    pdl_wait();
    pdl_trigger();
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= S) return;
    double tot = 0.0;
    for (long long i = item_ptr[j]; i < item_ptr[j + 1]; ++i) tot += partial[i];
    out[j] = tot;
}
// x_j <- max(0, x_j - lambda eta^k * (reduced step)_j); the reduced statistics follow the step in the buffer
__global__ void __launch_bounds__(256) k_update_from(long long S, const double* __restrict__ rbuf, double* __restrict__ x, DevState* st) {
    pdl_wait();
    pdl_trigger();
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j == 0) { st->prox = rbuf[S]; st->phi = rbuf[S + 1]; st->n_viol = (long long)rbuf[S + 2]; }
    if (j >= S) return;
    const double v = x[j] - st->relax * rbuf[j];
    x[j] = v < 0.0 ? 0.0 : v;
}

// |g|^2 (partial sums of k_combine) and c (partial sums of F2) in fixed order, then the `while loop` of Fig. 3
// on device scalars.  The step is
// b = beta (or beta / |g| with the normalised-gradient option).  Two-sided cost (Eq. 2 as printed):
//     chi^2(x - b g) = chi^2(x) - b |g|^2 + b^2 c   =>   accept  <=>  b c < |g|^2       (no pass per trial).
// One-sided cost option: chi^2 is piecewise quadratic, so every trial evaluates chi^2(x - b g) from d - b Dg, l - b Lg
// (a pass over the labelled rows' vectors, not over the matrix).  The accepted step (0 if none) goes to st->beta_acc;
// k_residual applies it.  One CTA.
__global__ void __launch_bounds__(1024)
k_select(DevState* st, const double* __restrict__ gpart, int n_gpart, const double* __restrict__ cpart, int n_part,
         const double* __restrict__ phipart, int n_phipart,
         long long n, const int16_t* __restrict__ rseg, const StructInfo* __restrict__ tab, const VoxBounds vb,
         const double* __restrict__ d, const double* __restrict__ l, const double* __restrict__ Dg, const double* __restrict__ Lg) {
    pdl_wait();
    pdl_trigger();
    __shared__ double sm[32];
    __shared__ double s_b;
    __shared__ int s_go;
    const double gg = block_sum(strided_sum(gpart, n_gpart), sm);
    const double cc = block_sum(strided_sum(cpart, n_part), sm);
    const double phi_x = block_sum(strided_sum(phipart, n_phipart), sm);   // chi^2(x) (partial sums of the pass that wrote p, q)
    const int flags = st->flags;
    if (!(flags & SF_ONE_SIDED)) {
        if (threadIdx.x == 0) {
            double acc = 0.0;
            if (gg > 0.0) {                                        // g == 0: nothing to reduce (reading R10)
                const double norm = (flags & SF_NORMALIZE_GRAD) ? sqrt(gg) : 1.0;
                const double aa = st->a;
                double bn = st->beta_next;
                long long s = st->s, tr = st->trials;
                const long long mt = st->max_trials;
                const int chk = st->accept_check;
                for (long long t = 0; t < mt; ++t) {
                    const double beta = bn;
                    bn *= aa; ++s; ++tr;
                    const double b = beta / norm;
                    // chi^2(x) - chi^2(x - b g) = b (|g|^2 - b c) exactly; Fig. 3 accepts iff chi^2(x - b g) < chi^2(x) as
                    // EVALUATED: a decrease below the fp64 resolution of chi^2(x) is not a decrease
                    const double dec = b * (gg - b * cc);
                    if (!chk || (dec > 0.0 && phi_x - dec < phi_x)) { acc = b; st->last_beta = beta; break; }
                }
                st->beta_next = bn; st->s = s; st->trials = tr;
            }
            st->beta_acc = acc; st->gg = gg; st->c = cc; st->phi = phi_x;
        }
        return;
    }
    // ---- one-sided cost: literal trials on the stored products
    if (threadIdx.x == 0) { s_go = gg > 0.0; st->gg = gg; st->c = cc; st->beta_acc = 0.0; }
    __syncthreads();
    if (!s_go) return;
    const double phi0 = cost_along(0.0, n, rseg, tab, vb, d, l, Dg, Lg, 1, sm);     // valid in thread 0
    const long long mt = st->max_trials;
    for (long long t = 0; t < mt; ++t) {
        __syncthreads();
        if (threadIdx.x == 0) {
            const double beta = st->beta_next;
            st->beta_next = beta * st->a; st->s += 1; st->trials += 1;
            s_b = (flags & SF_NORMALIZE_GRAD) ? beta / sqrt(gg) : beta;
        }
        __syncthreads();
        const double b = s_b;
        double phi = 0.0;
        const int chk = st->accept_check;
        if (chk) phi = cost_along(b, n, rseg, tab, vb, d, l, Dg, Lg, 1, sm);
        if (threadIdx.x == 0) {
            const int ok = !chk || phi < phi0;
            if (ok) { st->beta_acc = b; st->last_beta = (flags & SF_NORMALIZE_GRAD) ? b * sqrt(gg) : b; }
            s_go = !ok;
        }
        __syncthreads();
        if (!s_go) break;
    }
}

// Per active row: apply the accepted perturbation to the stored products (d' = d - beta Dg, l' = l - beta Lg) and
// per spot to the weights (x' = x - beta g); then, if `final`, the residuals of Fig. 2 in simultaneous form at x':
//   u_i = w^ r_dose/|D_i|^2 - LETmax w^ r_letd/|L_i - LETmax D_i|^2 ,  v_i = w^ r_dl/|L_i|^2 + w^ r_letd/|...|^2
// plus partial sums of the proximity, chi^2 and the violation count (fixed grid, fixed order); if not final
// (another reduction of Fig. 3 follows), the cost residuals p, q at x'.
__global__ void __launch_bounds__(ROW_THREADS)
k_residual(long long n, const int16_t* __restrict__ rseg, const StructInfo* __restrict__ tab, const VoxBounds vb, DevState* st,
           double* __restrict__ d, double* __restrict__ l, const double* __restrict__ Dg, const double* __restrict__ Lg,
           const double* __restrict__ nD, const double* __restrict__ nL, const double* __restrict__ nT,
           const GatherVec uv, const GatherVec pq, double* __restrict__ x, const double* __restrict__ g, long long S,
           double* __restrict__ part_prox, double* __restrict__ part_phi, long long* __restrict__ part_cnt,
           int use_beta, int final, int write_uv, uint8_t* __restrict__ live, int R) {
    pdl_wait();
    pdl_trigger();
    __shared__ double sm[ROW_THREADS / 32];
    __shared__ long long smc[ROW_THREADS / 32];
    const double beta = use_beta ? st->beta_acc : 0.0;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x, nth = (long long)gridDim.x * blockDim.x;
    const int lane = threadIdx.x & 31;
    if (beta != 0.0)
        for (long long j = tid; j < S; j += nth) x[j] = fma(-beta, g[j], x[j]);
    double prox = 0.0, phi = 0.0;
    long long cnt = 0;
    for (long long a0 = tid - lane; a0 < n; a0 += nth) {            // whole warps: the R rows of a block row sit in R neighbouring lanes
        const long long a = a0 + lane;
        const int sg = a < n ? rseg[a] : -1;                          // -1: padding row of a ragged block (no sets, no cost term)
        int nz = 0;
        if (sg >= 0) {
            double dv = d[a], lv = l[a];
            if (beta != 0.0) {
                dv = fma(-beta, Dg[a], dv);
                lv = fma(-beta, Lg[a], lv);
                d[a] = dv; l[a] = lv;
            }
            const StructInfo& T = tab[sg];
            const int f = T.flags;
            const double w = T.what;
            const RowBounds B = row_bounds(T, vb, a);
            if (!final) {
                double pv, qv;
                cost_residuals(f, w, B.dose_ref, B.dl_ref, st->flags & SF_ONE_SIDED, dv, lv, pv, qv);
                gv_store(pq, a, pv, qv);
                if (f & F_DOSE_REF) { const double e = B.dose_ref - dv; phi += w * e * e; }
                if (f & F_DL_REF) { const double e = B.dl_ref - lv; if (!((st->flags & SF_ONE_SIDED) && e > 0.0)) phi += w * e * e; }
            } else {
                double uu, vv;
                row_residual(T, B, st->flags & SF_ONE_SIDED, dv, lv, nD[a], nL[a], nT[a], uu, vv, cnt, prox, phi);
                if (write_uv) gv_store(uv, a, uu, vv);
                nz = (uu != 0.0) | (vv != 0.0);
            }
        }
        if (final && write_uv) {                                       // liveness byte of the block row (read by the back-projection)
            if (R >= 2) nz |= __shfl_xor_sync(0xffffffffu, nz, 1);
            if (R == 4) nz |= __shfl_xor_sync(0xffffffffu, nz, 2);
            if (a < n && (a % R) == 0) live[a / R] = (uint8_t)nz;
        }
    }
    if (!final) {                                                  // chi^2(x') for the next reduction's accept test
        const double q = block_sum(phi, sm);
        if (threadIdx.x == 0) part_phi[blockIdx.x] = q;
    }
    if (final) {
        const double p = block_sum(prox, sm);
        const double q = block_sum(phi, sm);
        // integer block sum
        long long c = cnt;
        for (int o = 16; o > 0; o >>= 1) c += __shfl_down_sync(0xffffffffu, c, o);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) smc[threadIdx.x >> 5] = c;
        __syncthreads();
        if (threadIdx.x == 0) {
            long long t = 0;
            for (int i = 0; i < ROW_THREADS / 32; ++i) t += smc[i];
            part_prox[blockIdx.x] = p; part_phi[blockIdx.x] = q; part_cnt[blockIdx.x] = t;
            if (blockIdx.x == 0 && write_uv) {                 // w_k = eta^k w: relax for this step
                st->relax = st->lambda * st->eta_pow;
                st->eta_pow *= st->eta;
                st->k += 1;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ block-sequential AMS (R23)
// Residual pass of ONE (kind, structure) block over its rows [rb, re) of the labelled list, at the x the block starts
// from: coefficient c_i = r_i / |a_i|^2 (0 where the norm is 0) into the gather vector (kind 0: D; 1: L; 2: L - LETmax D),
// the block's violated sets (integer atomics: order-independent) and partial sums of its proximity share.
__global__ void __launch_bounds__(ROW_THREADS)
k_block_residual(long long rb, long long re, int seg, int kind, const StructInfo* __restrict__ tab, const VoxBounds vb, DevState* st,
                 const double* __restrict__ d, const double* __restrict__ l, const double* __restrict__ nD,
                 const double* __restrict__ nL, const double* __restrict__ nT, const GatherVec uv,
                 double* __restrict__ part_prox) {
    pdl_wait();
    pdl_trigger();
    __shared__ double sm[ROW_THREADS / 32];
    __shared__ unsigned long long smc[ROW_THREADS / 32];
    const StructInfo& T = tab[seg];
    const double w = T.what;
    double prox = 0.0;
    unsigned long long cnt = 0;
    for (long long a = rb + (long long)blockIdx.x * blockDim.x + threadIdx.x; a < re; a += (long long)gridDim.x * blockDim.x) {
        const RowBounds B = row_bounds(T, vb, a);
        double r, nn;
        if (kind == 0) { r = slab_residual(d[a], B.dose_lo, B.dose_hi); nn = nD[a]; }
        else if (kind == 1) { r = slab_residual(l[a], B.dl_lo, B.dl_hi); nn = nL[a]; }
        else { const double val = l[a] - B.letd_max * d[a]; r = val > 0.0 ? val : 0.0; nn = nT[a]; }
        if (r != 0.0) ++cnt;
        double c = 0.0;
        if (nn > 0.0 && r != 0.0) { c = r / nn; prox += 0.5 * w * r * r / nn; }
        if (kind == 0) gv_store(uv, a, c, 0.0);
        else if (kind == 1) gv_store(uv, a, 0.0, c);
        else gv_store(uv, a, -B.letd_max * c, c);
    }
    const double p = block_sum(prox, sm);
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_down_sync(0xffffffffu, cnt, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) smc[threadIdx.x >> 5] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
        for (int i = 0; i < ROW_THREADS / 32; ++i) t += smc[i];
        part_prox[blockIdx.x] = p;
        if (t) atomicAdd((unsigned long long*)&st->n_viol, t);
    }
}

// Second stage of a block's transposed pass: x_j <- x_j - lambda eta^k min(w_s, 1) / m * (sum of the block's slots of
// spot j); block 0 also adds the block's proximity share (fixed order) to the sweep statistics.
__global__ void __launch_bounds__(256)
k_combine_block(long long S, const long long* __restrict__ slot_ptr, int seg, int n_seg, int H,
                const double* __restrict__ partial, double* __restrict__ x, DevState* st, double factor,
                const double* __restrict__ part_prox, int n_part) {
    pdl_wait();
    pdl_trigger();
    if (blockIdx.x == 0 && threadIdx.x < 32) {
        double p = 0.0;
        for (int i = threadIdx.x; i < n_part; i += 32) p += part_prox[i];
        p = warp_sum(p);
        if (threadIdx.x == 0) st->prox += p;
    }
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= S) return;
    const long long ib = slot_ptr[(j * n_seg + seg) * H], ie = slot_ptr[(j * n_seg + seg + 1) * H];
    if (ib == ie) return;
    double tot = 0.0;
    for (long long i = ib; i < ie; ++i) tot += partial[i];
    x[j] -= st->lambda * st->eta_pow * factor * tot;
}

// Start of a block-sequential sweep: the sweep statistics restart.
__global__ void k_sweep_begin(DevState* st) { pdl_wait(); pdl_trigger(); st->prox = 0.0; st->n_viol = 0; }

// End of a block-sequential sweep: clamp, w_{k+1} = eta * w_k, k <- k + 1.
__global__ void __launch_bounds__(256)
k_sweep_end(long long S, double* __restrict__ x, DevState* st) {
    pdl_wait();
    pdl_trigger();
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j < S && x[j] < 0.0) x[j] = 0.0;
    if (j == 0) { st->relax = st->lambda * st->eta_pow; st->eta_pow *= st->eta; st->k += 1; }
}

__global__ void __launch_bounds__(1024)
k_finalize_stats(DevState* st, const double* __restrict__ part_prox, const double* __restrict__ part_phi,
                 const long long* __restrict__ part_cnt, int n_part) {
    pdl_wait();
    pdl_trigger();
    __shared__ double sm[32];
    __shared__ long long smc[32];
    double p = 0.0, q = 0.0;
    long long c = 0;
    p = strided_sum(part_prox, n_part);
    q = strided_sum(part_phi, n_part);
    for (int i = threadIdx.x; i < n_part; i += blockDim.x) c += part_cnt[i];
    const double P = block_sum(p, sm);
    const double Q = block_sum(q, sm);
    for (int o = 16; o > 0; o >>= 1) c += __shfl_down_sync(0xffffffffu, c, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) smc[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long t = 0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += smc[i];
        st->prox = P; st->phi = Q; st->n_viol = t;
    }
}

}  // namespace fredopt
