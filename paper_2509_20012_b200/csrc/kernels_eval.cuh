// kernels_eval.cuh -- kernels of the calls outside the iteration (launched from passes.cu only): evaluation quantities
// (DVH / LVH / cDLVH, cDL30, Table 1), vector conversions, the streaming-read ceiling.
#pragma once
#include "fredopt_kernels.cuh"

namespace fredopt {

// ------------------------------------------------------------------------------------------ evaluation
// value of a voxel quantity from the stored products: 0 dose d, 1 cDL l, 2 LETd l/d (0 where d = 0)
__global__ void k_quantity(long long n, int quantity, const double* __restrict__ d, const double* __restrict__ l,
                           double* __restrict__ out) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n; a += (long long)gridDim.x * blockDim.x) {
        const double dv = d[a], lv = l[a];
        out[a] = quantity == 0 ? dv : quantity == 1 ? lv : (dv > 0.0 ? lv / dv : 0.0);
    }
}
// min, sum, max of n values in fixed order (one CTA): out[0..2]
__global__ void __launch_bounds__(1024)
k_value_stats(long long n, const double* __restrict__ v, double* __restrict__ out) {
    __shared__ double sm[32];
    double mn = INFINITY, mx = -INFINITY, sum = 0.0;
    for (long long a = threadIdx.x; a < n; a += blockDim.x) { const double t = v[a]; mn = fmin(mn, t); mx = fmax(mx, t); sum += t; }
    const double S = block_sum(sum, sm);
    for (int o = 16; o > 0; o >>= 1) { mn = fmin(mn, __shfl_down_sync(0xffffffffu, mn, o)); mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o)); }
    __shared__ double smn[32], smx[32];
    if ((threadIdx.x & 31) == 0) { smn[threadIdx.x >> 5] = mn; smx[threadIdx.x >> 5] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < (int)(blockDim.x >> 5); ++i) { mn = fmin(mn, smn[i]); mx = fmax(mx, smx[i]); }
        out[0] = mn; out[1] = S; out[2] = mx;
    }
}
// cnt[b] += 1 for the largest b with b * vmax / n_bins <= value (values below edge 0 are not counted)
__global__ void k_value_hist(long long n, const double* __restrict__ v, int n_bins, double vmax, unsigned long long* __restrict__ cnt) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n; a += (long long)gridDim.x * blockDim.x) {
        const double t = v[a];
        if (!(t >= 0.0)) continue;                       // edge 0 is 0
        double g = floor(t / vmax * (double)n_bins);
        int b = g >= (double)(n_bins - 1) ? n_bins - 1 : (int)g;
        while (b + 1 < n_bins && (double)(b + 1) * vmax / (double)n_bins <= t) ++b;
        while (b > 0 && (double)b * vmax / (double)n_bins > t) --b;
        atomicAdd(cnt + b, 1ULL);
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
// out[a] = {u[vox[a]], v[vox[a]]}   (voxel-indexed fp32 -> item-indexed fp64 pairs; a null input reads as 0)
__global__ void k_gather_uv(const float* __restrict__ u, const float* __restrict__ v, const int32_t* __restrict__ vox,
                            const GatherVec out, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int vx = vox[i];                                       // -1: padding row of a ragged block
        gv_store(out, i, (u && vx >= 0) ? (double)u[vx] : 0.0, (v && vx >= 0) ? (double)v[vx] : 0.0);
    }
}

// per-voxel values of one bound field (voxel-indexed fp32, NaN = the structure's scalar) -> row-indexed effective fp64 values;
// *bad |= 1 on an infinite value
__global__ void k_vb_fill(long long n_rows, const int32_t* __restrict__ vox, const int16_t* __restrict__ rseg,
                          const StructInfo* __restrict__ tab, int field, const float* __restrict__ values, double* __restrict__ out,
                          int* __restrict__ bad) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n_rows; a += (long long)gridDim.x * blockDim.x) {
        const int sg = rseg[a];
        if (sg < 0) { out[a] = 0.0; continue; }
        const StructInfo& T = tab[sg];
        const double sc = field == VB_DOSE_LO ? T.dose_lo : field == VB_DOSE_HI ? T.dose_hi : field == VB_DL_LO ? T.dl_lo
                        : field == VB_DL_HI ? T.dl_hi : field == VB_LETD_MAX ? T.letd_max : field == VB_DOSE_REF ? T.dose_ref : T.dl_ref;
        const float v = values[vox[a]];
        if (isinf(v)) *bad = 1;
        out[a] = isnan(v) ? sc : (double)v;
    }
}
// lo <= hi on every row (comparisons with NaN = absent are false)
__global__ void k_vb_check(long long n_rows, const int16_t* __restrict__ rseg, const StructInfo* __restrict__ tab, const VoxBounds vb,
                           int* __restrict__ bad) {
    for (long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x; a < n_rows; a += (long long)gridDim.x * blockDim.x) {
        const int sg = rseg[a];
        if (sg < 0) continue;
        const RowBounds B = row_bounds(tab[sg], vb, a);
        if (B.dose_lo > B.dose_hi || B.dl_lo > B.dl_hi) *bad = 1;
    }
}

// read-only streaming sum (practical ceiling of a 100%-read pass): 8 independent 128-bit loads per thread
__global__ void __launch_bounds__(256)
k_stream_read(const int4* __restrict__ p, long long n16, int* __restrict__ sink) {
    const long long base = (long long)blockIdx.x * 2048 + threadIdx.x;
    int4 v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const long long i = base + u * 256;
        v[u] = i < n16 ? ld_stream_i4((const int32_t*)(p + i)) : make_int4(0, 0, 0, 0);
    }
    int acc = 0;
#pragma unroll
    for (int u = 0; u < 8; ++u) acc += v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
    if (acc == 0x7fffffff) *sink = acc;      // never true in practice; keeps the loads alive
}

}  // namespace fredopt
