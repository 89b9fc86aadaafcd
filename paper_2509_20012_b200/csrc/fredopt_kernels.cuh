// fredopt_kernels.cuh -- the hot kernels of the superiorized feasibility-seeking iteration (sm_100a).
//
// Passes of one iteration:
//   k_forward    d = D x, l = L x   over a row list (warp per row, 128-bit streamed index/value loads, fp64
//                accumulation, shuffle reduction).  Rows read only the value arrays their structure needs.
//   k_transpose  out_j = sum_i D_ij cD_i + L_ij cL_i   over the stored CSR of the transposes (CTA per spot,
//                per-structure segments, no atomics, fixed-order reduction) with the gradient / update+clamp
//                epilogues fused.
//   k_select     |g|^2, c = sum w^ (Dg)^2 + w^ (Lg)^2, the accept loop of Fig. 3 on device scalars, x' = x - beta g.
//   k_residual   d' = d - beta Dg, l' = l - beta Lg, residuals / violations of Fig. 2 -> u, v, partial sums.
// All vectors and accumulators are fp64; matrix values fp32; indices int32; offsets int64.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fredopt {

constexpr int FWD_THREADS = 256;
constexpr int FWD_WARPS = FWD_THREADS / 32;
constexpr int TR_THREADS = 256;
constexpr int MAX_PARTIALS = 1184;          // 148 SMs x 8 resident CTAs of 256 threads
constexpr int ROW_THREADS = 256;

// flags of a structure
enum : int { F_DOSE_SLAB = 1, F_DL_SLAB = 2, F_LETD = 4, F_DOSE_REF = 8, F_DL_REF = 16 };

struct StructInfo {
    double w, what;
    double dose_lo, dose_hi, dl_lo, dl_hi, letd_max, dose_ref, dl_ref;
    int flags, pad;
    unsigned long long part, n_sets, n_zero, rows, nnz;   // participating sets, declared sets, zero-norm sets, rows, nnz
};

struct SegCoef { double scaleD, shiftD, scaleL, shiftL; };   // coefficient = scale * (vec[a] - shift)

struct DevState {
    double lambda, beta0, a, eta;
    double beta_next, eta_pow, relax, last_beta, beta_acc;
    double phi, prox, gg, c, W;
    long long k, s, trials, n_viol, max_trials;
    long long n_sets, n_zero;
    int accept_check, pad;
};

// ------------------------------------------------------------------------------------------ loads
// streamed arrays (index / value): read once, keep them out of L1 so that L1 holds the gathered vector
__device__ __forceinline__ int4 ld_stream_i4(const int32_t* p) {
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ float4 ld_stream_f4(const float* p) {
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// fixed-order block sum; result valid in thread 0.  `sm` holds >= blockDim.x/32 doubles.
__device__ __forceinline__ double block_sum(double v, double* sm) {
    v = warp_sum(v);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = blockDim.x >> 5;
    __syncthreads();
    if (l == 0) sm[w] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0) for (int i = 0; i < nw; ++i) r += sm[i];
    return r;
}

// ------------------------------------------------------------------------------------------ forward
struct RowList {
    long long n;                 // rows in the list
    const long long* start;      // [n] offset of the row in the padded arrays (multiple of 4)
    const int32_t* len;          // [n] padded length (multiple of 4)
    const int32_t* seg;          // [n] segment (structure - 1), or nullptr = segment 0
    const int32_t* vox;          // [n] voxel index of the row
};

enum : int { EPI_STORE = 0, EPI_CPART = 1, EPI_F32VOX = 2 };

__device__ __forceinline__ void fma4(double& acc, const float4& a, double x0, double x1, double x2, double x3) {
    acc = fma((double)a.x, x0, acc);
    acc = fma((double)a.y, x1, acc);
    acc = fma((double)a.z, x2, acc);
    acc = fma((double)a.w, x3, acc);
}

// One warp per row, rows r = warp, warp + W, ... (static mapping: deterministic partial sums).
// mode[seg]: bit 0 = read valD, bit 1 = read valL.
template <int EPI>
__global__ void __launch_bounds__(FWD_THREADS)
k_forward(RowList rl, const uint8_t* __restrict__ mode, const int32_t* __restrict__ col,
          const float* __restrict__ vD, const float* __restrict__ vL, const double* __restrict__ x,
          double* __restrict__ oD, double* __restrict__ oL,               // EPI_STORE / EPI_CPART: list-indexed
          const StructInfo* __restrict__ tab, double* __restrict__ cpart,  // EPI_CPART
          float* __restrict__ fD, float* __restrict__ fL, int letd_out)    // EPI_F32VOX: voxel-indexed
{
    const int lane = threadIdx.x & 31;
    const long long warp0 = (long long)blockIdx.x * FWD_WARPS + (threadIdx.x >> 5);
    const long long nwarps = (long long)gridDim.x * FWD_WARPS;
    double csum = 0.0;
    for (long long r = warp0; r < rl.n; r += nwarps) {
        const long long s = rl.start[r];
        const int L = rl.len[r];
        const int sg = rl.seg ? rl.seg[r] : 0;
        const int m = mode[sg];
        double aD = 0.0, aL = 0.0;
        if (m != 0) {
            const int32_t* cp = col + s;
            const float* dp = vD + s;
            const float* lp = vL + s;
            int p = lane * 4;
            for (; p + 128 < L; p += 256) {
                const int4 c0 = ld_stream_i4(cp + p), c1 = ld_stream_i4(cp + p + 128);
                float4 d0, d1, l0, l1;
                if (m & 1) { d0 = ld_stream_f4(dp + p); d1 = ld_stream_f4(dp + p + 128); }
                if (m & 2) { l0 = ld_stream_f4(lp + p); l1 = ld_stream_f4(lp + p + 128); }
                const double x0 = __ldg(x + c0.x), x1 = __ldg(x + c0.y), x2 = __ldg(x + c0.z), x3 = __ldg(x + c0.w);
                const double y0 = __ldg(x + c1.x), y1 = __ldg(x + c1.y), y2 = __ldg(x + c1.z), y3 = __ldg(x + c1.w);
                if (m & 1) { fma4(aD, d0, x0, x1, x2, x3); fma4(aD, d1, y0, y1, y2, y3); }
                if (m & 2) { fma4(aL, l0, x0, x1, x2, x3); fma4(aL, l1, y0, y1, y2, y3); }
            }
            if (p < L) {
                const int4 c0 = ld_stream_i4(cp + p);
                float4 d0, l0;
                if (m & 1) d0 = ld_stream_f4(dp + p);
                if (m & 2) l0 = ld_stream_f4(lp + p);
                const double x0 = __ldg(x + c0.x), x1 = __ldg(x + c0.y), x2 = __ldg(x + c0.z), x3 = __ldg(x + c0.w);
                if (m & 1) fma4(aD, d0, x0, x1, x2, x3);
                if (m & 2) fma4(aL, l0, x0, x1, x2, x3);
            }
            aD = warp_sum(aD);
            aL = warp_sum(aL);
        }
        if (lane == 0) {
            if (EPI == EPI_F32VOX) {
                const int v = rl.vox[r];
                if (fD) fD[v] = (float)aD;
                if (fL) fL[v] = letd_out ? (aD > 0.0 ? (float)(aL / aD) : 0.0f) : (float)aL;
            } else {
                oD[r] = aD;
                oL[r] = aL;
                if (EPI == EPI_CPART) {
                    const StructInfo& T = tab[sg];
                    if (T.flags & F_DOSE_REF) csum += T.what * aD * aD;
                    if (T.flags & F_DL_REF) csum += T.what * aL * aL;
                }
            }
        }
    }
    if (EPI == EPI_CPART) {
        __shared__ double sm[FWD_WARPS];
        // lane 0 of each warp carries that warp's sum; other lanes carry 0
        const double t = block_sum(csum, sm);
        if (threadIdx.x == 0) cpart[blockIdx.x] = t;
    }
}

// ------------------------------------------------------------------------------------------ transposed
enum : int { TEPI_F32 = 0, TEPI_GRAD = 1, TEPI_UPDATE = 2 };

// One CTA per spot j.  The spot's entries are stored per structure segment (t_ptr[j*n_seg + s]), columns =
// compact active-row indices in ascending order; entry coefficient = scale_s * (vec[a] - shift_s).
template <int EPI>
__global__ void __launch_bounds__(TR_THREADS)
k_transpose(int n_seg, const long long* __restrict__ t_ptr, const int32_t* __restrict__ t_col,
            const float* __restrict__ tD, const float* __restrict__ tL, const uint8_t* __restrict__ mode,
            const SegCoef* __restrict__ coef, const double* __restrict__ vecD, const double* __restrict__ vecL,
            double* __restrict__ g_out,                    // TEPI_GRAD
            double* __restrict__ x, const DevState* __restrict__ st,   // TEPI_UPDATE
            float* __restrict__ f_out)                     // TEPI_F32
{
    __shared__ double sm[TR_THREADS / 32];
    const long long j = blockIdx.x;
    double acc = 0.0;
    for (int sg = 0; sg < n_seg; ++sg) {
        const int m = mode[sg];
        if (m == 0) continue;
        const long long b = t_ptr[j * n_seg + sg], e = t_ptr[j * n_seg + sg + 1];
        if (b == e) continue;
        const SegCoef cf = coef[sg];
        double aD = 0.0, aL = 0.0;
        long long p = b + threadIdx.x * 4;
        for (; p + TR_THREADS * 4 < e; p += TR_THREADS * 8) {
            const int4 c0 = ld_stream_i4(t_col + p), c1 = ld_stream_i4(t_col + p + TR_THREADS * 4);
            if (m & 1) {
                const float4 a0 = ld_stream_f4(tD + p), a1 = ld_stream_f4(tD + p + TR_THREADS * 4);
                const double s = cf.shiftD;
                fma4(aD, a0, __ldg(vecD + c0.x) - s, __ldg(vecD + c0.y) - s, __ldg(vecD + c0.z) - s, __ldg(vecD + c0.w) - s);
                fma4(aD, a1, __ldg(vecD + c1.x) - s, __ldg(vecD + c1.y) - s, __ldg(vecD + c1.z) - s, __ldg(vecD + c1.w) - s);
            }
            if (m & 2) {
                const float4 a0 = ld_stream_f4(tL + p), a1 = ld_stream_f4(tL + p + TR_THREADS * 4);
                const double s = cf.shiftL;
                fma4(aL, a0, __ldg(vecL + c0.x) - s, __ldg(vecL + c0.y) - s, __ldg(vecL + c0.z) - s, __ldg(vecL + c0.w) - s);
                fma4(aL, a1, __ldg(vecL + c1.x) - s, __ldg(vecL + c1.y) - s, __ldg(vecL + c1.z) - s, __ldg(vecL + c1.w) - s);
            }
        }
        if (p < e) {
            const int4 c0 = ld_stream_i4(t_col + p);
            if (m & 1) {
                const float4 a0 = ld_stream_f4(tD + p);
                const double s = cf.shiftD;
                fma4(aD, a0, __ldg(vecD + c0.x) - s, __ldg(vecD + c0.y) - s, __ldg(vecD + c0.z) - s, __ldg(vecD + c0.w) - s);
            }
            if (m & 2) {
                const float4 a0 = ld_stream_f4(tL + p);
                const double s = cf.shiftL;
                fma4(aL, a0, __ldg(vecL + c0.x) - s, __ldg(vecL + c0.y) - s, __ldg(vecL + c0.z) - s, __ldg(vecL + c0.w) - s);
            }
        }
        acc += cf.scaleD * aD + cf.scaleL * aL;
    }
    const double tot = block_sum(acc, sm);
    if (threadIdx.x == 0) {
        if (EPI == TEPI_GRAD) g_out[j] = tot;
        else if (EPI == TEPI_UPDATE) {
            const double v = x[j] - st->relax * tot;          // x <- x' - lambda eta^k * sum w^ (r/|a|^2) a
            x[j] = v < 0.0 ? 0.0 : v;                          // clamp
        } else f_out[j] = (float)tot;
    }
}

// ------------------------------------------------------------------------------------------ scalar kernels
__global__ void k_set_params(DevState* st, double lambda, double beta0, double a, double eta, long long max_trials,
                             int accept_check, int latch) {
    st->lambda = lambda;
    st->eta = eta;
    st->max_trials = max_trials;
    st->accept_check = accept_check;
    if (latch) { st->beta0 = beta0; st->a = a; st->beta_next = beta0; st->eta_pow = 1.0; }
}

// |g|^2 and c by fixed-order sums, then the `while loop` of Fig. 3 on scalars:
// chi^2(x - beta g) = chi^2(x) - beta |g|^2 + beta^2 c   =>   accept  <=>  beta c < |g|^2.
// Then x <- x - beta g.  One CTA.
__global__ void __launch_bounds__(1024)
k_select(DevState* st, const double* __restrict__ g, double* __restrict__ x, long long S,
         const double* __restrict__ cpart, int n_part) {
    __shared__ double sm[32];
    __shared__ double s_beta;
    double a = 0.0;
    for (long long j = threadIdx.x; j < S; j += blockDim.x) a = fma(g[j], g[j], a);
    const double gg = block_sum(a, sm);
    double c = 0.0;
    for (int i = threadIdx.x; i < n_part; i += blockDim.x) c += cpart[i];
    const double cc = block_sum(c, sm);
    if (threadIdx.x == 0) {
        double acc = 0.0;
        if (gg > 0.0) {                                        // g == 0: nothing to reduce (reading R10)
            const double aa = st->a;
            double bn = st->beta_next;
            long long s = st->s, tr = st->trials;
            const long long mt = st->max_trials;
            const int chk = st->accept_check;
            for (long long t = 0; t < mt; ++t) {
                const double beta = bn;
                bn *= aa; ++s; ++tr;
                if (!chk || beta * cc < gg) { acc = beta; st->last_beta = beta; break; }
            }
            st->beta_next = bn; st->s = s; st->trials = tr;
        }
        st->beta_acc = acc; st->gg = gg; st->c = cc;
        s_beta = acc;
    }
    __syncthreads();
    const double beta = s_beta;
    if (beta != 0.0)
        for (long long j = threadIdx.x; j < S; j += blockDim.x) x[j] = fma(-beta, g[j], x[j]);
}

// signed residual of a hyperslab lo <= val <= hi (NaN = absent): upper violations > 0, lower < 0
__device__ __forceinline__ double slab_residual(double val, double lo, double hi) {
    if (val > hi) return val - hi;      // false when hi is NaN
    if (val < lo) return val - lo;      // false when lo is NaN
    return 0.0;
}

// Per active row: apply the accepted perturbation to the stored products (d' = d - beta Dg, l' = l - beta Lg),
// then, if `final`, the residuals of Fig. 2 in simultaneous form at that point:
//   u_i = w^ r_dose/|D_i|^2 - LETmax w^ r_letd/|L_i - LETmax D_i|^2 ,  v_i = w^ r_dl/|L_i|^2 + w^ r_letd/|...|^2
// plus partial sums of the proximity, chi^2 and the violation count (fixed grid, fixed order).
__global__ void __launch_bounds__(ROW_THREADS)
k_residual(long long n, const int32_t* __restrict__ seg, const StructInfo* __restrict__ tab, DevState* st,
           double* __restrict__ d, double* __restrict__ l, const double* __restrict__ Dg, const double* __restrict__ Lg,
           const double* __restrict__ nD, const double* __restrict__ nL, const double* __restrict__ nT,
           double* __restrict__ u, double* __restrict__ v,
           double* __restrict__ part_prox, double* __restrict__ part_phi, long long* __restrict__ part_cnt,
           int use_beta, int final, int write_uv) {
    __shared__ double sm[ROW_THREADS / 32];
    __shared__ long long smc[ROW_THREADS / 32];
    const double beta = use_beta ? st->beta_acc : 0.0;
    double prox = 0.0, phi = 0.0;
    long long cnt = 0;
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n; a += (long long)gridDim.x * blockDim.x) {
        double dv = d[a], lv = l[a];
        if (beta != 0.0) {
            dv = fma(-beta, Dg[a], dv);
            lv = fma(-beta, Lg[a], lv);
            d[a] = dv; l[a] = lv;
        }
        if (!final) continue;
        const StructInfo& T = tab[seg[a]];
        const int f = T.flags;
        const double w = T.what;
        double cD = 0.0, cL = 0.0, cT = 0.0;
        if (f & (F_DOSE_SLAB)) {
            const double r = slab_residual(dv, T.dose_lo, T.dose_hi);
            if (r != 0.0) { ++cnt; const double nn = nD[a]; if (nn > 0.0) { cD = w * r / nn; prox += 0.5 * w * r * r / nn; } }
        }
        if (f & (F_DL_SLAB)) {
            const double r = slab_residual(lv, T.dl_lo, T.dl_hi);
            if (r != 0.0) { ++cnt; const double nn = nL[a]; if (nn > 0.0) { cL = w * r / nn; prox += 0.5 * w * r * r / nn; } }
        }
        if (f & (F_LETD)) {
            const double val = lv - T.letd_max * dv;
            if (val > 0.0) { ++cnt; const double nn = nT[a]; if (nn > 0.0) { cT = w * val / nn; prox += 0.5 * w * val * val / nn; } }
        }
        if (f & F_DOSE_REF) { const double e = T.dose_ref - dv; phi += w * e * e; }
        if (f & F_DL_REF) { const double e = T.dl_ref - lv; phi += w * e * e; }
        if (write_uv) {
            u[a] = (f & F_LETD) ? cD - T.letd_max * cT : cD;     // row of the LETd set is L_i - LETmax D_i
            v[a] = cL + cT;
        }
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

__global__ void __launch_bounds__(1024)
k_finalize_stats(DevState* st, const double* __restrict__ part_prox, const double* __restrict__ part_phi,
                 const long long* __restrict__ part_cnt, int n_part) {
    __shared__ double sm[32];
    __shared__ long long smc[32];
    double p = 0.0, q = 0.0;
    long long c = 0;
    for (int i = threadIdx.x; i < n_part; i += blockDim.x) { p += part_prox[i]; q += part_phi[i]; c += part_cnt[i]; }
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

// ------------------------------------------------------------------------------------------ small helpers
__global__ void k_f32_to_f64(const float* __restrict__ in, double* __restrict__ out, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        out[i] = (double)in[i];
}
__global__ void k_f64_to_f32(const double* __restrict__ in, float* __restrict__ out, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        out[i] = (float)in[i];
}
// out[a] = (double) in[vox[a]]   (voxel-indexed fp32 -> list-indexed fp64)
__global__ void k_gather_f32_to_f64(const float* __restrict__ in, const int32_t* __restrict__ vox,
                                    double* __restrict__ out, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        out[i] = (double)in[vox[i]];
}

// read-only streaming sum (practical ceiling of a 100%-read pass)
__global__ void __launch_bounds__(512)
k_stream_read(const int4* __restrict__ p, long long n16, int* __restrict__ sink) {
    int acc = 0;
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (; i + 3 * stride < n16; i += 4 * stride) {
        const int4 a = ld_stream_i4((const int32_t*)(p + i)), b = ld_stream_i4((const int32_t*)(p + i + stride));
        const int4 c = ld_stream_i4((const int32_t*)(p + i + 2 * stride)), d = ld_stream_i4((const int32_t*)(p + i + 3 * stride));
        acc += a.x ^ a.y ^ a.z ^ a.w ^ b.x ^ b.y ^ b.z ^ b.w ^ c.x ^ c.y ^ c.z ^ c.w ^ d.x ^ d.y ^ d.z ^ d.w;
    }
    for (; i < n16; i += stride) { const int4 a = ld_stream_i4((const int32_t*)(p + i)); acc += a.x ^ a.y ^ a.z ^ a.w; }
    if (acc == 0x7fffffff) *sink = acc;      // never true in practice; keeps the loads alive
}

}  // namespace fredopt
