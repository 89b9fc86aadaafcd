// fredopt_kernels.cuh -- the hot kernels of the superiorized feasibility-seeking iteration (sm_100a).
//
// Storage: the labelled rows are kept as BLOCK ROWS of R = 1, 2 or 4 consecutive voxels of one
// structure over the union of their column patterns (neighbouring voxels see almost the same spots): one stored index and
// one gathered weight serve R values, in both orientations -- an ENTRY is one (block row, spot) pair with R values per matrix.
//
// Passes of one iteration:
//   k_forward    d = D x, l = L x over a list of work items (one item = one block row; one warp per item,
//                round-robin, 128-bit streamed index/value loads kept out of L1, fp64 accumulation, shuffle
//                reduction).  A row reads only the value arrays its structure needs.  Epilogues: store d, l
//                (+ the cost residuals p, q of Eq. 2), the quadratic coefficient c of the accept test, the residuals /
//                violations of Fig. 2 with their statistics (pure feasibility-seeking), or fp32 dose / LETd per voxel.
//   k_transpose  out_j = sum_i D_ij u_i + L_ij v_i over the stored CSR of the transposes (one item = at most
//                TR_ITEM_MAX entries of one (structure, spot) run; one warp per item; every item writes its
//                partial sum to a fixed slot: no atomics, no fences).
//   k_combine    adds the slots of every spot in slot order and runs the gradient / update+clamp epilogue.
//   k_select     |g|^2, c = sum w^ (Dg)^2 + w^ (Lg)^2 and the accept loop of Fig. 3 on device scalars.
//   k_residual   d' = d - beta Dg, l' = l - beta Lg, x' = x - beta g, residuals / violations of Fig. 2 -> u, v,
//                partial sums of proximity, cost and violation count.
// All vectors and accumulators are fp64; matrix values fp32; indices 16-bit where they fit, else int32; offsets int64.
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <stdio.h>

namespace fredopt {

constexpr int FWD_THREADS = 256;
constexpr int FWD_WARPS = FWD_THREADS / 32;
constexpr int MAX_PARTIALS = 2368;          // 148 SMs x 16 CTAs: upper bound of any partial-sum grid
constexpr int ROW_THREADS = 256;
#ifndef TR_ITEM_MAX_ENTRIES
#define TR_ITEM_MAX_ENTRIES 2048   /* measured on configs[3]: 1024 -> -3 %, 4096 -> -0.3 %; on configs[1]: 4096 -> -7 % */
#endif
constexpr int TR_ITEM_MAX = TR_ITEM_MAX_ENTRIES;   // entries per transposed work item (multiple of 128)
#ifndef FWD_U1
#define FWD_U1 6   /* 128-entry chunks in flight per trip for rows that read one matrix ... */
#endif
#ifndef FWD_U3
#define FWD_U3 4   /* ... and for rows that read both (measured: 6/4 beats 4/4 by 2 %, 8/4 and 6/3 are slower) */
#endif
#ifndef FWD_MIN_CTAS_PER_SM
#define FWD_MIN_CTAS_PER_SM 4
#endif
// spare (zeroed) elements behind every stored index array: tr_item_live loads the indices of a trip one trip ahead and may run
// up to U + 1 chunks of 128 entries past the last item; such words are never used
constexpr size_t IDX_SLACK = 1024;
static_assert(128 * (FWD_U1 + 1) <= IDX_SLACK && 128 * (FWD_U3 + 1) <= IDX_SLACK, "index look-ahead stays inside the spare elements");
constexpr int FWD_MIN_CTAS = FWD_MIN_CTAS_PER_SM;   // resident CTAs per SM the item kernels are compiled for (4: 64 registers)

// flags of a structure
enum : int { F_DOSE_SLAB = 1, F_DL_SLAB = 2, F_LETD = 4, F_DOSE_REF = 8, F_DL_REF = 16 };
enum : int { SF_NORMALIZE_GRAD = 1, SF_ONE_SIDED = 2 };

struct DevState;
// cost residuals of Eq. (2) at (d, l): p = 2 w^ (d - Dref), q = 2 w^ (l - cDLref) [one-sided: only where l > cDLref]
__device__ __forceinline__ void cost_residuals(int f, double w, double dref, double lref, int one_sided, double dv, double lv,
                                               double& p, double& q) {
    p = (f & F_DOSE_REF) ? 2.0 * w * (dv - dref) : 0.0;
    q = (f & F_DL_REF) ? 2.0 * w * (lv - lref) : 0.0;
    if (one_sided && q < 0.0) q = 0.0;
}

struct StructInfo {
    double w, what;
    double dose_lo, dose_hi, dl_lo, dl_hi, letd_max, dose_ref, dl_ref;
    int flags, pad;
    unsigned long long part, n_sets, n_zero, rows, nnz;   // participating sets, declared sets, zero-norm sets, rows, nnz
    unsigned long long entries;                           // stored entries (union patterns of the structure's block rows)
    unsigned long long part_kind[3];                      // participating sets per kind: dose slab, cDL slab, LETd
};

struct DevState {
    double lambda, beta0, a, eta;
    double beta_next, eta_pow, relax, last_beta, beta_acc;
    double phi, prox, gg, c, W;
    long long k, s, trials, n_viol, max_trials;
    long long n_sets, n_zero;
    int accept_check;
    int flags;                 // bit 0: step along g/|g| (R9 option); bit 1: one-sided cDL cost (R11 option)
};

// Per-voxel bounds and references (bounds "defined for each point in the image space"; Eq. (2), PAPER.md:207-210:
// Dref_i, cDLref_i): per field an optional row-indexed array of EFFECTIVE values (the voxel's own value, else the structure's
// scalar); a null pointer = the structure's scalar everywhere.  Which kinds / cost terms a row has stays with its structure.
enum : int { VB_DOSE_LO = 0, VB_DOSE_HI, VB_DL_LO, VB_DL_HI, VB_LETD_MAX, VB_DOSE_REF, VB_DL_REF, VB_N };
struct VoxBounds { const double* f[VB_N]; };
struct RowBounds { double dose_lo, dose_hi, dl_lo, dl_hi, letd_max, dose_ref, dl_ref; };
__device__ __forceinline__ RowBounds row_bounds(const StructInfo& T, const VoxBounds& vb, long long r) {
    RowBounds b;
    b.dose_lo = vb.f[VB_DOSE_LO] ? vb.f[VB_DOSE_LO][r] : T.dose_lo;
    b.dose_hi = vb.f[VB_DOSE_HI] ? vb.f[VB_DOSE_HI][r] : T.dose_hi;
    b.dl_lo = vb.f[VB_DL_LO] ? vb.f[VB_DL_LO][r] : T.dl_lo;
    b.dl_hi = vb.f[VB_DL_HI] ? vb.f[VB_DL_HI][r] : T.dl_hi;
    b.letd_max = vb.f[VB_LETD_MAX] ? vb.f[VB_LETD_MAX][r] : T.letd_max;
    b.dose_ref = vb.f[VB_DOSE_REF] ? vb.f[VB_DOSE_REF][r] : T.dose_ref;
    b.dl_ref = vb.f[VB_DL_REF] ? vb.f[VB_DL_REF][r] : T.dl_ref;
    return b;
}

// One work item: `len` VALUES per matrix (multiple of 4) starting at value `start` (multiple of 4) of the value arrays,
// i.e. len / R entries starting at entry start / R of the index array; `seg` & 0xFF = structure - 1 (selects which value
// arrays are read).  Forward items (one block row) carry the number of real rows of the block (1..R; the last block of a
// structure may be ragged) in bits 8-10; transposed items carry the 65536-block group of their 16-bit block indices in
// seg >> 8.  16 bytes: fetched with one 128-bit load.
struct __align__(16) Item {
    long long start;
    int32_t len;
    int32_t seg;
};

// Gather vector of a transposed pass, item-indexed, kept in two layouts: runs that need both matrices gather one
// 16-byte pair per entry; runs that need one matrix gather from the dense 8-byte array (four rows per 32-byte sector).
struct GatherVec {
    double2* pair;   // {coefficient of D_i, coefficient of L_i}
    double* cD;
    double* cL;
};
__device__ __forceinline__ void gv_store(const GatherVec& g, long long a, double vd, double vl) {
    double2 v; v.x = vd; v.y = vl;
    g.pair[a] = v; g.cD[a] = vd; g.cL[a] = vl;
}

// Programmatic dependent launch (griddepcontrol, sm_90+): the kernels of one iteration are launched with programmatic
// stream serialization, so a kernel's CTAs may be scheduled while its predecessor drains.  pdl_wait() returns when the
// predecessor grid has completed and its writes are visible (a no-op for an ordinary launch); pdl_trigger() lets the
// successor start being scheduled.  Every kernel waits before it touches anything another kernel writes, and triggers
// only after its own wait, so kernel N+2 can never run ahead of kernel N.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ------------------------------------------------------------------------------------------ checked build
// -DFREDOPT_CHECKED (python paper_2509_20012_b200/build.py -DFREDOPT_CHECKED): every load of the item kernels -- streamed
// indices and values, item descriptors, gathered weights / coefficients, liveness bytes -- is checked against the extents of
// the live plans' device allocations and traps with a message when it lies outside all of them.  Slow; for the tests only
// (compute-sanitizer is closed on this pool: profiles/r02_sanitizer.md).
#ifdef FREDOPT_CHECKED
struct ChkRange { const char* b; const char* e; };
constexpr int CHK_MAX = 2048;
static __device__ ChkRange g_chk[CHK_MAX];
static __device__ int g_chk_n;
static __device__ __noinline__ void chk_fail(const void* p, int bytes, int site) {
    printf("fredopt checked build: load of %d bytes at %p lies outside every allocation of a plan (site %d, block %d, thread %d)\n", bytes, p, site,
           (int)blockIdx.x, (int)threadIdx.x);
    __trap();
}
__device__ __forceinline__ void chk(const void* p, int bytes, int site) {
    const char* a = (const char*)p;
    const int n = g_chk_n;
    for (int i = 0; i < n; ++i)
        if (a >= g_chk[i].b && a + bytes <= g_chk[i].e) return;
    chk_fail(p, bytes, site);
}
// this translation unit's copy of the table
static inline void chk_upload_tu(const ChkRange* h, int n) {
    cudaMemcpyToSymbol(g_chk, h, (size_t)n * sizeof(ChkRange));
    cudaMemcpyToSymbol(g_chk_n, &n, sizeof(int));
}
#else
#define chk(p, bytes, site) ((void)0)
#endif

// ------------------------------------------------------------------------------------------ loads
// Timing experiments (results are WRONG on purpose; profiles/r02_ceilings.md): -DEXP_NO_GATHER makes the gathered value from the
// index without a load, -DEXP_NO_CVT skips the fp32 -> fp64 conversion, -DEXP_NO_FMA replaces the fp64 multiply-add by an xor.
#ifdef EXP_NO_GATHER
#define FWD_GATHER(x, c) __hiloint2double(0x3ff00000, (c))
#else
__device__ __forceinline__ double fwd_gather(const double* __restrict__ x, int c) { chk(x + c, 8, 8); return __ldg(x + c); }
#define FWD_GATHER(x, c) fwd_gather((x), (c))
#endif
// streamed arrays (index / value): read once, keep them out of L1 so that L1 holds the gathered vector
__device__ __forceinline__ int4 ld_stream_i4(const int32_t* p) {
    int4 r;
    chk(p, 16, 1);
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
// four consecutive stored values of a matrix as fp32: stored as fp32 (one 128-bit load) or, with the 16-bit value option of
// fredopt_create_options, as IEEE half (one 64-bit load; half -> float is exact)
__device__ __forceinline__ float4 ld_stream_f4(const __half* p) {
    unsigned int lo, hi;
    chk(p, 8, 2);
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(lo), "=r"(hi) : "l"(p));
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&lo)), b = __half22float2(*reinterpret_cast<const __half2*>(&hi));
    return make_float4(a.x, a.y, b.x, b.y);
}
__device__ __forceinline__ float4 ld_stream_f4(const float* p) {
    float4 r;
    chk(p, 16, 2);
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
// C consecutive stored indices starting at index position i (a multiple of C): 16-bit form (+ `add`) or 32-bit form.
// C = 4 / R is the number of entries a lane's 128-bit value load covers.
template <bool I16, int C>
__device__ __forceinline__ void ld_idx(const void* __restrict__ base, long long i, int add, int (&c)[C]) {
    chk((const char*)base + i * (I16 ? 2 : 4), C * (I16 ? 2 : 4), 3);
    if (I16) {
        const uint16_t* p = (const uint16_t*)base + i;
        if (C == 4) {
            unsigned int lo, hi;
            asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(lo), "=r"(hi) : "l"(p));
            c[0] = (int)(lo & 0xFFFFu) + add; c[1 % C] = (int)(lo >> 16) + add; c[2 % C] = (int)(hi & 0xFFFFu) + add; c[3 % C] = (int)(hi >> 16) + add;
        } else if (C == 2) {
            unsigned int lo;
            asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(lo) : "l"(p));
            c[0] = (int)(lo & 0xFFFFu) + add; c[1 % C] = (int)(lo >> 16) + add;
        } else {
            unsigned short lo;
            asm volatile("ld.global.nc.L1::no_allocate.u16 %0, [%1];" : "=h"(lo) : "l"(p));
            c[0] = (int)lo + add;
        }
    } else {
        const int32_t* p = (const int32_t*)base + i;
        if (C == 4) {
            const int4 v = ld_stream_i4(p);
            c[0] = v.x; c[1 % C] = v.y; c[2 % C] = v.z; c[3 % C] = v.w;
        } else if (C == 2) {
            int a, b;
            asm volatile("ld.global.nc.L1::no_allocate.v2.s32 {%0,%1}, [%2];" : "=r"(a), "=r"(b) : "l"(p));
            c[0] = a; c[1 % C] = b;
        } else {
            int a;
            asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(a) : "l"(p));
            c[0] = a;
        }
    }
}
// the same indices as loaded (16-bit form: two per word), unpacked where they are used: tr_item_live keeps the indices of the
// next trip in registers
template <bool I16, int C> struct IdxRaw { unsigned int w[I16 ? (C + 1) / 2 : C]; };
template <bool I16, int C>
__device__ __forceinline__ void ld_idx_raw(const void* __restrict__ base, long long i, IdxRaw<I16, C>& r) {
    chk((const char*)base + i * (I16 ? 2 : 4), C * (I16 ? 2 : 4), 4);
    if (I16) {
        const uint16_t* p = (const uint16_t*)base + i;
        if (C == 4) {
            asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(r.w[0]), "=r"(r.w[(C + 1) / 2 - 1]) : "l"(p));
        } else if (C == 2) {
            asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(r.w[0]) : "l"(p));
        } else {
            unsigned short lo;
            asm volatile("ld.global.nc.L1::no_allocate.u16 %0, [%1];" : "=h"(lo) : "l"(p));
            r.w[0] = lo;
        }
    } else {
        const int32_t* p = (const int32_t*)base + i;
        if (C == 4) {
            asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.w[0]), "=r"(r.w[1 % C]), "=r"(r.w[2 % C]), "=r"(r.w[3 % C]) : "l"(p));
        } else if (C == 2) {
            asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(r.w[0]), "=r"(r.w[1 % C]) : "l"(p));
        } else {
            asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(r.w[0]) : "l"(p));
        }
    }
}
template <bool I16, int C>
__device__ __forceinline__ int idx_get(const IdxRaw<I16, C>& r, int j, int add) {
    if (I16) {
        const unsigned int w = r.w[j / 2];
        return (int)((j & 1) ? (w >> 16) : (w & 0xFFFFu)) + add;
    }
    return (int)r.w[j];
}
__device__ __forceinline__ Item ld_item(const Item* p) {
    chk(p, 16, 5);
    const int4 v = __ldg((const int4*)p);
    Item it;
    it.start = (long long)(((unsigned long long)(unsigned)v.y << 32) | (unsigned)v.x);
    it.len = v.z;
    it.seg = v.w;
    return it;
}
// R consecutive fp64 coefficients starting at element R * b of a gathered vector (cached: neighbouring entries reuse lines)
template <int R>
__device__ __forceinline__ void ld_coef(const double* __restrict__ v, int b, double (&g)[R]) {
#ifdef EXP_NO_GATHER
    for (int k = 0; k < R; ++k) g[k] = __hiloint2double(0x3ff00000, b + k);
    return;
#endif
    chk(v + (long long)R * b, 8 * R, 6);
    if (R == 1) g[0] = __ldg(v + b);
    else if (R == 2) { const double2 t = __ldg((const double2*)v + b); g[0] = t.x; g[1 % R] = t.y; }
    else {   // 32 bytes, 32-byte aligned: one 256-bit load (sm_100+)
        double a0, a1, a2, a3;
        asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a0), "=d"(a1), "=d"(a2), "=d"(a3) : "l"(v + 4 * (long long)b));
        g[0] = a0; g[1 % R] = a1; g[2 % R] = a2; g[3 % R] = a3;
    }
}
// R consecutive {coefficient of D_i, coefficient of L_i} pairs starting at pair R * b
template <int R>
__device__ __forceinline__ void ld_coef_pair(const double2* __restrict__ v, int b, double (&gd)[R], double (&gl)[R]) {
#ifdef EXP_NO_GATHER
    for (int k = 0; k < R; ++k) { gd[k] = __hiloint2double(0x3ff00000, b + k); gl[k] = __hiloint2double(0x3ff00000, b - k); }
    return;
#endif
    chk(v + (long long)R * b, 16 * R, 7);
    if (R == 1) { const double2 t = __ldg(v + b); gd[0] = t.x; gl[0] = t.y; }
    else {
#pragma unroll
        for (int h = 0; h < R / 2; ++h) {   // 32 bytes (two pairs) per 256-bit load
            double a0, a1, a2, a3;
            asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a0), "=d"(a1), "=d"(a2), "=d"(a3) : "l"(v + (long long)R * b + 2 * h));
            gd[(2 * h) % R] = a0; gl[(2 * h) % R] = a1; gd[(2 * h + 1) % R] = a2; gl[(2 * h + 1) % R] = a3;
        }
    }
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

__device__ __forceinline__ float f4_get(const float4& a, int i) { return i == 0 ? a.x : i == 1 ? a.y : i == 2 ? a.z : a.w; }
// a stored value as fp64 and the multiply-add of the matrix passes (the experiments above replace them)
__device__ __forceinline__ double f2d(float v) {
#ifdef EXP_NO_CVT
    return __hiloint2double(0x3ff00000, (int)__float_as_uint(v));
#else
    return (double)v;
#endif
}
__device__ __forceinline__ double fma_op(double a, double b, double c) {
#ifdef EXP_NO_FMA
    return __longlong_as_double(__double_as_longlong(a) ^ __double_as_longlong(b) ^ __double_as_longlong(c));
#else
    return fma(a, b, c);
#endif
}

// signed residual of a hyperslab lo <= val <= hi (NaN = absent): upper violations > 0, lower < 0
__device__ __forceinline__ double slab_residual(double val, double lo, double hi) {
    if (val > hi) return val - hi;      // false when hi is NaN
    if (val < lo) return val - lo;      // false when lo is NaN
    return 0.0;
}

// Residuals of Fig. 2 for one labelled row at (dv, lv) in simultaneous form: the coefficients of D_i and L_i in the step,
//   u_i = w^ r_dose/|D_i|^2 - LETmax w^ r_letd/|L_i - LETmax D_i|^2 ,  v_i = w^ r_dl/|L_i|^2 + w^ r_letd/|...|^2 ,
// and the row's share of the violated-set count, the proximity and chi^2.
__device__ __forceinline__ void row_residual(const StructInfo& S_, const RowBounds& T, int one_sided, double dv, double lv, double nD,
                                             double nL, double nT, double& u, double& v, long long& cnt, double& prox, double& phi) {
    const int f = S_.flags;
    const double w = S_.what;
    double cD = 0.0, cL = 0.0, cT = 0.0;
    if (f & F_DOSE_SLAB) {
        const double r = slab_residual(dv, T.dose_lo, T.dose_hi);
        if (r != 0.0) { ++cnt; if (nD > 0.0) { cD = w * r / nD; prox += 0.5 * w * r * r / nD; } }
    }
    if (f & F_DL_SLAB) {
        const double r = slab_residual(lv, T.dl_lo, T.dl_hi);
        if (r != 0.0) { ++cnt; if (nL > 0.0) { cL = w * r / nL; prox += 0.5 * w * r * r / nL; } }
    }
    if (f & F_LETD) {
        const double val = lv - T.letd_max * dv;
        if (val > 0.0) { ++cnt; if (nT > 0.0) { cT = w * val / nT; prox += 0.5 * w * val * val / nT; } }
    }
    if (f & F_DOSE_REF) { const double e = T.dose_ref - dv; phi += w * e * e; }
    if (f & F_DL_REF) { const double e = T.dl_ref - lv; if (!(one_sided && e > 0.0)) phi += w * e * e; }
    u = (f & F_LETD) ? cD - T.letd_max * cT : cD;     // row of the LETd set is L_i - LETmax D_i
    v = cL + cT;
}

// fixed-order block sum of an integer; result valid in thread 0
__device__ __forceinline__ long long block_sum_ll(long long c, long long* smc) {
    for (int o = 16; o > 0; o >>= 1) c += __shfl_down_sync(0xffffffffu, c, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) smc[threadIdx.x >> 5] = c;
    __syncthreads();
    long long t = 0;
    if (threadIdx.x == 0) for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += smc[i];
    return t;
}

// what the residual epilogue of the forward kernel needs (EPI_RESID)
struct ResidArgs {
    const double *nD, *nL, *nT;          // squared norms per labelled row
    GatherVec uv;                        // out: step coefficients (null pointers: statistics only)
    double *part_prox, *part_phi;        // out: per-CTA partial sums
    long long* part_cnt;
    DevState* st;                        // relax = lambda eta^k, eta^k and k advance when uv is written
    uint8_t* live;                       // out: per block row, 1 iff one of its rows has a non-zero step coefficient (with uv)
};

// ------------------------------------------------------------------------------------------ work distribution
// The items of a pass are dealt to the warps of a persistent grid (one CTA per resident slot) from a queue: the first two
// items of a warp are static (warp, warp + W), the others come from an integer counter, longest items first -- a warp that
// finishes early takes more work, so the pass ends when the work ends, not when the unluckiest warp of a static deal does.
// Which warp computes an item never changes a result: an item's sum is formed by one warp in a fixed lane order and stored
// to a place that belongs to the item (row, slot, per-item partial sums), so the passes stay bitwise reproducible.  The last
// warp to leave resets the queue for the next launch (launches of a plan are serialised on its stream).
struct WorkQueue {
    unsigned int next;           // items handed out beyond the static ones
    unsigned int done;           // warps that have left
};
__device__ __forceinline__ void queue_leave(WorkQueue* q, int lane, unsigned int n_warps) {
    if (lane == 0) {
        const unsigned int old = atomicAdd(&q->done, 1u);
        if (old == n_warps - 1) { q->next = 0u; q->done = 0u; }          // everyone else has stopped fetching
    }
}
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

// ------------------------------------------------------------------------------------------ forward
enum : int { EPI_STORE = 0, EPI_STORE_PQ = 1, EPI_CPART = 2, EPI_F32VOX = 3, EPI_RESID = 4 };

// <D_i, x> and / or <L_i, x> of the R rows of one block row by one warp.  M: bit 0 = D, bit 1 = L.  Lv values per matrix
// (multiple of 4) starting at value v0: a lane's 128-bit load holds C = 4 / R entries (R values each); inside every chunk of
// 128 values the entries are stored interleaved so that the j-th gather of the warp covers CONSECUTIVE entries (few lines of
// x per instruction).  U chunks per trip (6 for a single matrix, 4 for both): up to 12 independent vector loads per lane in
// flight before the first gather.
template <int M, int R, bool I16, typename VT>
__device__ __forceinline__ void fwd_row(const void* __restrict__ cbase, long long v0, const VT* __restrict__ dp,
                                        const VT* __restrict__ lp, int Lv, int lane, const double* __restrict__ x,
                                        double (&aD)[R], double (&aL)[R]) {
    constexpr int C = 4 / R;
    constexpr int U = (M == 3) ? FWD_U3 : FWD_U1;
    const long long i0 = v0 / R;                 // first stored index of the block row
    int p = lane * 4;
    for (; p + 128 * (U - 1) < Lv; p += 128 * U) {
        int c[U][C];
        float4 d[U], l[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            ld_idx<I16, C>(cbase, i0 + (p + 128 * u) / R, 0, c[u]);
            if (M & 1) d[u] = ld_stream_f4(dp + p + 128 * u);
            if (M & 2) l[u] = ld_stream_f4(lp + p + 128 * u);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            double xv[C];
#pragma unroll
            for (int j = 0; j < C; ++j) xv[j] = FWD_GATHER(x, c[u][j]);
#pragma unroll
            for (int j = 0; j < C; ++j)
#pragma unroll
                for (int k = 0; k < R; ++k) {
                    if (M & 1) aD[k] = fma_op(f2d(f4_get(d[u], j * R + k)), xv[j], aD[k]);
                    if (M & 2) aL[k] = fma_op(f2d(f4_get(l[u], j * R + k)), xv[j], aL[k]);
                }
        }
    }
    if (p < Lv) {   // remainder (fewer than U chunks): ONE predicated trip, all loads in flight together; a lane without
                    // an entry behaves like padding (column 0, value 0)
        int c[U - 1][C];
        float4 d[U - 1], l[U - 1];
#pragma unroll
        for (int u = 0; u < U - 1; ++u) {
            const bool ok = p + 128 * u < Lv;
            if (ok) ld_idx<I16, C>(cbase, i0 + (p + 128 * u) / R, 0, c[u]);
            else {
#pragma unroll
                for (int j = 0; j < C; ++j) c[u][j] = 0;
            }
            if (M & 1) d[u] = ok ? ld_stream_f4(dp + p + 128 * u) : make_float4(0.f, 0.f, 0.f, 0.f);
            if (M & 2) l[u] = ok ? ld_stream_f4(lp + p + 128 * u) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < U - 1; ++u) {
            if (p + 128 * u < Lv) {
                double xv[C];
#pragma unroll
                for (int j = 0; j < C; ++j) xv[j] = FWD_GATHER(x, c[u][j]);
#pragma unroll
                for (int j = 0; j < C; ++j)
#pragma unroll
                    for (int k = 0; k < R; ++k) {
                        if (M & 1) aD[k] = fma_op(f2d(f4_get(d[u], j * R + k)), xv[j], aD[k]);
                        if (M & 2) aL[k] = fma_op(f2d(f4_get(l[u], j * R + k)), xv[j], aL[k]);
                    }
            }
        }
    }
}

// One warp per item (block row) from the work queue (items in longest-first order; item_blk[e] = block row of item e, or null
// = e).  The descriptor of the next item is fetched while the current one is processed.  mode[seg]: bit 0 = read valD, bit 1 =
// read valL.  Row r = R * b + k (k < rows of the block) indexes every per-row array; partial sums of the epilogues (c, chi^2,
// proximity, count) are stored per block row and added in a fixed order by the kernel that consumes them.
template <int EPI, int R, bool I16, typename VT>
__global__ void __launch_bounds__(FWD_THREADS, FWD_MIN_CTAS)
k_forward(long long n, const Item* __restrict__ items, const int32_t* __restrict__ item_blk, WorkQueue* __restrict__ wq,
          const int32_t* __restrict__ vox, const uint8_t* __restrict__ mode,
          const void* __restrict__ col, const VT* __restrict__ vD, const VT* __restrict__ vL,
          const double* __restrict__ x,
          double* __restrict__ oD, double* __restrict__ oL,                // EPI_STORE*, EPI_CPART, EPI_RESID: row-indexed
          const GatherVec pq,                                              // EPI_STORE_PQ: cost residuals (Eq. 2)
          const StructInfo* __restrict__ tab, const VoxBounds vb, double* __restrict__ cpart,  // EPI_STORE_PQ / EPI_CPART: per block row
          const DevState* __restrict__ st,                                 // EPI_STORE_PQ (cost form)
          float* __restrict__ fD, float* __restrict__ fL, int letd_out,    // EPI_F32VOX: voxel-indexed
          const ResidArgs ra)                                              // EPI_RESID: residual / violation epilogue (a7)
{
    const int lane = threadIdx.x & 31;
    const int nwarps = gridDim.x * FWD_WARPS, ni = (int)n;      // items < 2^31
    int e0 = blockIdx.x * FWD_WARPS + (threadIdx.x >> 5), e1 = e0 + nwarps;
    if (e0 < ni) prefetch_l1(items + e0);                       // static data: touched before the dependency wait
    pdl_wait();
    pdl_trigger();
    while (e0 < ni) {
        const Item it = ld_item(items + e0);
        const int blk = item_blk ? item_blk[e0] : e0;
        unsigned int e2 = 0;
        if (wq && lane == 0) e2 = atomicAdd(&wq->next, 1u);     // in flight while this item is processed
        if (e1 < ni) { prefetch_l1(items + e1); if (item_blk) prefetch_l1(item_blk + e1); }
        const long long b = blk;
        const int seg = it.seg & 0xFF, nrow = (it.seg >> 8) & 7;
        const int m = mode[seg];
        double aD[R], aL[R];
#pragma unroll
        for (int k = 0; k < R; ++k) { aD[k] = 0.0; aL[k] = 0.0; }
        if (m == 3) fwd_row<3, R, I16>(col, it.start, vD + it.start, vL + it.start, it.len, lane, x, aD, aL);
        else if (m == 1) fwd_row<1, R, I16>(col, it.start, vD + it.start, (const VT*)nullptr, it.len, lane, x, aD, aL);
        else if (m == 2) fwd_row<2, R, I16>(col, it.start, (const VT*)nullptr, vL + it.start, it.len, lane, x, aD, aL);
#pragma unroll
        for (int k = 0; k < R; ++k) {
            if (m & 1) aD[k] = warp_sum(aD[k]);
            if (m & 2) aL[k] = warp_sum(aL[k]);
        }
        if (lane == 0) {
            double csum = 0.0, rprox = 0.0, rphi = 0.0;
            long long rcnt = 0;
            int nzb = 0;
#pragma unroll
            for (int k = 0; k < R; ++k) {
                if (k >= nrow) break;
                const long long r = b * R + k;
                const double dv = aD[k], lv = aL[k];
                if (EPI == EPI_F32VOX) {
                    const int v = vox[r];
                    if (fD) fD[v] = (float)dv;
                    if (fL) fL[v] = letd_out ? (dv > 0.0 ? (float)(lv / dv) : 0.0f) : (float)lv;
                } else {
                    oD[r] = dv;
                    oL[r] = lv;
                    if (EPI == EPI_STORE_PQ) {      // p_i = 2 w^ (d_i - Dref), q_i = 2 w^ (l_i - cDLref): grad chi^2 = D^T p + L^T q
                        const StructInfo& T = tab[seg];
                        const int one_sided = st->flags & SF_ONE_SIDED;
                        const double dref = vb.f[VB_DOSE_REF] ? vb.f[VB_DOSE_REF][r] : T.dose_ref;
                        const double lref = vb.f[VB_DL_REF] ? vb.f[VB_DL_REF][r] : T.dl_ref;
                        double pv, qv;
                        cost_residuals(T.flags, T.what, dref, lref, one_sided, dv, lv, pv, qv);
                        gv_store(pq, r, pv, qv);
                        // the row's share of chi^2(x) (Eq. 2): the accept test of Fig. 3 compares against it
                        if (T.flags & F_DOSE_REF) { const double e = dref - dv; csum += T.what * e * e; }
                        if (T.flags & F_DL_REF) { const double e = lref - lv; if (!(one_sided && e > 0.0)) csum += T.what * e * e; }
                    }
                    if (EPI == EPI_CPART) {
                        const StructInfo& T = tab[seg];
                        if (T.flags & F_DOSE_REF) csum += T.what * dv * dv;
                        if (T.flags & F_DL_REF) csum += T.what * lv * lv;
                    }
                    if (EPI == EPI_RESID) {         // residuals / violations of Fig. 2 at x, in the epilogue of the fused pass
                        double u, v;
                        row_residual(tab[seg], row_bounds(tab[seg], vb, r), ra.st->flags & SF_ONE_SIDED, dv, lv, ra.nD[r], ra.nL[r], ra.nT[r], u, v,
                                     rcnt, rprox, rphi);
                        if (ra.uv.pair) gv_store(ra.uv, r, u, v);
                        nzb |= (u != 0.0) | (v != 0.0);
                    }
                }
            }
            if (EPI == EPI_CPART || EPI == EPI_STORE_PQ) cpart[b] = csum;
            if (EPI == EPI_RESID) {
                ra.part_prox[b] = rprox; ra.part_phi[b] = rphi; ra.part_cnt[b] = rcnt;
                if (ra.uv.pair) ra.live[b] = (uint8_t)nzb;
            }
        }
        e0 = e1;
        e1 = wq ? 2 * nwarps + (int)__shfl_sync(0xffffffffu, e2, 0) : e1 + nwarps;      // no queue: static round-robin
    }
    if (wq) queue_leave(wq, lane, (unsigned int)nwarps);
    if (EPI == EPI_RESID && blockIdx.x == 0 && threadIdx.x == 0 && ra.uv.pair) {   // w_k = eta^k w: relax for this step
        ra.st->relax = ra.st->lambda * ra.st->eta_pow;
        ra.st->eta_pow *= ra.st->eta;
        ra.st->k += 1;
    }
}

// Short rows of the full row set (R = 1; at most 4*G entries, G = 4, 8 or 16): G lanes per row, 32/G rows per warp at a time,
// one 128-bit load per lane and array, shuffle reduction inside the lane group.  Rows of one length class are stored back to
// back, so the warp's loads are contiguous.  fp32 voxel-indexed outputs only (fredopt_dose_let / fredopt_spmv_forward over
// all rows).
template <int G, bool I16>
__global__ void __launch_bounds__(FWD_THREADS)
k_forward_short(long long n, const Item* __restrict__ items, const int32_t* __restrict__ vox, int m,
                const void* __restrict__ col, const float* __restrict__ vD, const float* __restrict__ vL,
                const double* __restrict__ x, float* __restrict__ fD, float* __restrict__ fL, int letd_out)
{
    constexpr int RPW = 32 / G;                       // rows per warp and trip
    const int lane = threadIdx.x & 31, t = lane % G, grp = lane / G;
    const long long nwarps = (long long)gridDim.x * FWD_WARPS;
    for (long long base = ((long long)blockIdx.x * FWD_WARPS + (threadIdx.x >> 5)) * RPW; base < n; base += nwarps * RPW) {
        const long long r = base + grp;
        double aD = 0.0, aL = 0.0;
        if (r < n) {
            const Item it = ld_item(items + r);
            if (4 * t < it.len) {
                const long long p = it.start + 4 * t;
                int c[4];
                ld_idx<I16, 4>(col, p, 0, c);
                const double x0 = __ldg(x + c[0]), x1 = __ldg(x + c[1]), x2 = __ldg(x + c[2]), x3 = __ldg(x + c[3]);
                if (m & 1) { const float4 a = ld_stream_f4(vD + p); aD = fma((double)a.x, x0, aD); aD = fma((double)a.y, x1, aD); aD = fma((double)a.z, x2, aD); aD = fma((double)a.w, x3, aD); }
                if (m & 2) { const float4 a = ld_stream_f4(vL + p); aL = fma((double)a.x, x0, aL); aL = fma((double)a.y, x1, aL); aL = fma((double)a.z, x2, aL); aL = fma((double)a.w, x3, aL); }
            }
        }
#pragma unroll
        for (int o = G / 2; o > 0; o >>= 1) {
            aD += __shfl_down_sync(0xffffffffu, aD, o, G);
            aL += __shfl_down_sync(0xffffffffu, aL, o, G);
        }
        if (t == 0 && r < n) {
            const int v = vox[r];
            if (fD) fD[v] = (float)aD;
            if (fL) fL[v] = letd_out ? (aD > 0.0 ? (float)(aL / aD) : 0.0f) : (float)aL;
        }
    }
}

// ------------------------------------------------------------------------------------------ transposed
enum : int { TEPI_F32 = 0, TEPI_GRAD = 1, TEPI_UPDATE = 2 };

// sum over one item of D_ij cD[i] + L_ij cL[i] by one warp: an entry is one (spot run, block row b) pair with R values per
// matrix and gathers the R coefficients of rows R b .. R b + R - 1 with one vector load (the gathered vectors are L2 / L1
// resident; entries of a run ascend in b, so neighbouring lanes gather neighbouring elements)
template <int M, int R, bool I16, typename VT>
__device__ __forceinline__ double tr_item(const void* __restrict__ cbase, long long v0, int add, const VT* __restrict__ dp,
                                          const VT* __restrict__ lp, int Lv, int lane, const GatherVec& gv) {
    constexpr int C = 4 / R;
    constexpr int U = (M == 3) ? FWD_U3 : FWD_U1;
    const double2* __restrict__ vec = gv.pair;
    const double* __restrict__ vs = (M == 2) ? gv.cL : gv.cD;
    const long long i0 = v0 / R;
    double aD = 0.0, aL = 0.0;
    int p = lane * 4;
#define TR_CONSUME(u)                                                                                     \
    _Pragma("unroll") for (int j = 0; j < C; ++j) {                                                        \
        if (M == 3) {                                                                                      \
            double gd[R], gl[R];                                                                           \
            ld_coef_pair<R>(vec, c[u][j], gd, gl);                                                         \
            _Pragma("unroll") for (int k = 0; k < R; ++k) {                                                \
                aD = fma_op(f2d(f4_get(d[u], j * R + k)), gd[k], aD);                                      \
                aL = fma_op(f2d(f4_get(l[u], j * R + k)), gl[k], aL);                                      \
            }                                                                                              \
        } else {                                                                                           \
            double g[R];                                                                                   \
            ld_coef<R>(vs, c[u][j], g);                                                                    \
            _Pragma("unroll") for (int k = 0; k < R; ++k) {                                                \
                if (M == 1) aD = fma_op(f2d(f4_get(d[u], j * R + k)), g[k], aD);                           \
                else aL = fma_op(f2d(f4_get(l[u], j * R + k)), g[k], aL);                                  \
            }                                                                                              \
        }                                                                                                  \
    }
    for (; p + 128 * (U - 1) < Lv; p += 128 * U) {
        int c[U][C];
        float4 d[U], l[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            ld_idx<I16, C>(cbase, i0 + (p + 128 * u) / R, add, c[u]);
            if (M & 1) d[u] = ld_stream_f4(dp + p + 128 * u);
            if (M & 2) l[u] = ld_stream_f4(lp + p + 128 * u);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) { TR_CONSUME(u) }
    }
    if (p < Lv) {   // remainder: one predicated trip (see fwd_row)
        int c[U - 1][C];
        float4 d[U - 1], l[U - 1];
#pragma unroll
        for (int u = 0; u < U - 1; ++u) {
            const bool ok = p + 128 * u < Lv;
            if (ok) ld_idx<I16, C>(cbase, i0 + (p + 128 * u) / R, add, c[u]);
            else {
#pragma unroll
                for (int j = 0; j < C; ++j) c[u][j] = 0;
            }
            if (M & 1) d[u] = ok ? ld_stream_f4(dp + p + 128 * u) : make_float4(0.f, 0.f, 0.f, 0.f);
            if (M & 2) l[u] = ok ? ld_stream_f4(lp + p + 128 * u) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < U - 1; ++u) {
            if (p + 128 * u < Lv) { TR_CONSUME(u) }
        }
    }
#undef TR_CONSUME
    return aD + aL;
}

// The same sum where most coefficients are zero (the back-projection of Fig. 2 touches a row only when its test fires,
// PAPER.md:129-146; after a few dozen iterations most sets are satisfied): live[b] != 0 iff block row b has a non-zero
// coefficient (written by the residual pass that wrote the coefficients).  A lane streams its 16 bytes of values per matrix and
// gathers only where one of its C entries is live; every skipped term is an exact zero, so the sum has the same bits.  The
// indices are needed BEFORE the values: those of a trip are loaded one trip ahead (a word or two per chunk and lane) and the
// liveness bytes (L1-resident) are looked up at the start of the trip.
template <int M, int R, bool I16, typename VT>
__device__ __forceinline__ double tr_item_live(const void* __restrict__ cbase, long long v0, int add, const VT* __restrict__ dp,
                                               const VT* __restrict__ lp, int Lv, int lane, const GatherVec& gv,
                                               const uint8_t* __restrict__ live) {
    constexpr int C = 4 / R;
    constexpr int U = (M == 3) ? FWD_U3 : FWD_U1;
    const double2* __restrict__ vec = gv.pair;
    const double* __restrict__ vs = (M == 2) ? gv.cL : gv.cD;
    const long long i0 = v0 / R;
    double aD = 0.0, aL = 0.0;
    int p = lane * 4;
#define TRL_CONSUME(cc, u)                                                                                \
    _Pragma("unroll") for (int j = 0; j < C; ++j) {                                                        \
        if ((lv >> ((u) * C + j)) & 1u) {                                                                  \
            const int b = (idx_get<I16, C>(cc[u], j, add));                                                \
            if (M == 3) {                                                                                  \
                double gd[R], gl[R];                                                                       \
                ld_coef_pair<R>(vec, b, gd, gl);                                                           \
                _Pragma("unroll") for (int k = 0; k < R; ++k) {                                            \
                    aD = fma_op(f2d(f4_get(d[u], j * R + k)), gd[k], aD);                                  \
                    aL = fma_op(f2d(f4_get(l[u], j * R + k)), gl[k], aL);                                  \
                }                                                                                          \
            } else {                                                                                       \
                double g[R];                                                                               \
                ld_coef<R>(vs, b, g);                                                                      \
                _Pragma("unroll") for (int k = 0; k < R; ++k) {                                            \
                    if (M == 1) aD = fma_op(f2d(f4_get(d[u], j * R + k)), g[k], aD);                       \
                    else aL = fma_op(f2d(f4_get(l[u], j * R + k)), g[k], aL);                              \
                }                                                                                          \
            }                                                                                              \
        }                                                                                                  \
    }
    IdxRaw<I16, C> cn[U];                        // the indices of the next trip
#pragma unroll
    for (int u = 0; u < U; ++u) ld_idx_raw<I16, C>(cbase, i0 + (p + 128 * u) / R, cn[u]);
    for (; p + 128 * (U - 1) < Lv; p += 128 * U) {
        IdxRaw<I16, C> c[U];
        float4 d[U], l[U];
        unsigned int lv = 0u;                    // bit u * C + j: entry j of chunk u is live
#pragma unroll
        for (int u = 0; u < U; ++u) {
            c[u] = cn[u];
#pragma unroll
            for (int j = 0; j < C; ++j) { const int bb = (idx_get<I16, C>(c[u], j, add)); chk(live + bb, 1, 9); lv |= (__ldg(live + bb) ? 1u : 0u) << (u * C + j); }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const bool any = (lv >> (u * C)) & ((1u << C) - 1u);
            if (M & 1) d[u] = any ? ld_stream_f4(dp + p + 128 * u) : make_float4(0.f, 0.f, 0.f, 0.f);
            if (M & 2) l[u] = any ? ld_stream_f4(lp + p + 128 * u) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) ld_idx_raw<I16, C>(cbase, i0 + (p + 128 * (U + u)) / R, cn[u]);
#pragma unroll
        for (int u = 0; u < U; ++u) { TRL_CONSUME(c, u) }
    }
    if (p < Lv) {   // remainder: one predicated trip; a lane beyond the item's end holds foreign indices and uses none of them
        float4 d[U - 1], l[U - 1];
        unsigned int lv = 0u;
#pragma unroll
        for (int u = 0; u < U - 1; ++u) {
            if (p + 128 * u < Lv) {
#pragma unroll
                for (int j = 0; j < C; ++j) { const int bb = (idx_get<I16, C>(cn[u], j, add)); chk(live + bb, 1, 9); lv |= (__ldg(live + bb) ? 1u : 0u) << (u * C + j); }
            }
        }
#pragma unroll
        for (int u = 0; u < U - 1; ++u) {
            const bool any = (lv >> (u * C)) & ((1u << C) - 1u);
            if (M & 1) d[u] = any ? ld_stream_f4(dp + p + 128 * u) : make_float4(0.f, 0.f, 0.f, 0.f);
            if (M & 2) l[u] = any ? ld_stream_f4(lp + p + 128 * u) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < U - 1; ++u) { TRL_CONSUME(cn, u) }
    }
#undef TRL_CONSUME
    return aD + aL;
}

// One warp per item from the work queue; items are in longest-first order (ties in (structure, spot) order, so the warps of
// a CTA mostly work on neighbouring spots of one structure and share L1 lines of the gather vector).  Item e stores its
// partial sum in slot item_slot[e]; k_combine adds the slots of every spot in slot order.  No floating-point atomics, no
// fences: the result does not depend on the schedule.
template <int R, bool I16, bool LIVE, typename VT>
__global__ void __launch_bounds__(FWD_THREADS, FWD_MIN_CTAS)
k_transpose(long long n, const Item* __restrict__ items, const int32_t* __restrict__ item_slot, WorkQueue* __restrict__ wq,
            const uint8_t* __restrict__ mode, const void* __restrict__ t_col, const VT* __restrict__ tD,
            const VT* __restrict__ tL, const GatherVec vec, double* __restrict__ partial,
            const uint8_t* __restrict__ live)          // LIVE: liveness byte per block row (tr_item_live)
{
    const int lane = threadIdx.x & 31;
    const int nwarps = gridDim.x * FWD_WARPS, ni = (int)n;
    int e0 = blockIdx.x * FWD_WARPS + (threadIdx.x >> 5), e1 = e0 + nwarps;
    if (e0 < ni) prefetch_l1(items + e0);
    pdl_wait();
    pdl_trigger();
    while (e0 < ni) {
        const Item it = ld_item(items + e0);
        unsigned int e2 = 0;
        if (wq && lane == 0) e2 = atomicAdd(&wq->next, 1u);
        if (e1 < ni) prefetch_l1(items + e1);
        const int m = mode[it.seg & 0xFF];
        const int add = (it.seg >> 8) << 16;              // 16-bit form: the run's group of 65536 block rows
        double tot = 0.0;
        if (LIVE) {
            if (m == 3) tot = tr_item_live<3, R, I16>(t_col, it.start, add, tD + it.start, tL + it.start, it.len, lane, vec, live);
            else if (m == 1) tot = tr_item_live<1, R, I16>(t_col, it.start, add, tD + it.start, (const VT*)nullptr, it.len, lane, vec, live);
            else if (m == 2) tot = tr_item_live<2, R, I16>(t_col, it.start, add, (const VT*)nullptr, tL + it.start, it.len, lane, vec, live);
        } else {
            if (m == 3) tot = tr_item<3, R, I16>(t_col, it.start, add, tD + it.start, tL + it.start, it.len, lane, vec);
            else if (m == 1) tot = tr_item<1, R, I16>(t_col, it.start, add, tD + it.start, (const VT*)nullptr, it.len, lane, vec);
            else if (m == 2) tot = tr_item<2, R, I16>(t_col, it.start, add, (const VT*)nullptr, tL + it.start, it.len, lane, vec);
        }
        if (m) tot = warp_sum(tot);
        if (lane == 0) partial[item_slot[e0]] = tot;
        e0 = e1;
        e1 = wq ? 2 * nwarps + (int)__shfl_sync(0xffffffffu, e2, 0) : e1 + nwarps;
    }
    if (wq) queue_leave(wq, lane, (unsigned int)nwarps);
}

// Measurement only (FREDOPT_OPT_TIME_PASSES): the values a back-projection with these liveness bytes NEEDS -- entries of the
// items whose block row is live, times R values, times the matrices the item's structure reads -- added to out[0].
template <int R, bool I16>
__global__ void __launch_bounds__(FWD_THREADS)
k_count_live(long long n, const Item* __restrict__ items, const uint8_t* __restrict__ mode, const void* __restrict__ t_col,
             const uint8_t* __restrict__ live, unsigned long long* __restrict__ out) {
    const int lane = threadIdx.x & 31;
    const long long nwarps = (long long)gridDim.x * FWD_WARPS;
    unsigned long long tot = 0;
    for (long long e = (long long)blockIdx.x * FWD_WARPS + (threadIdx.x >> 5); e < n; e += nwarps) {
        const Item it = ld_item(items + e);
        const int m = mode[it.seg & 0xFF], add = (it.seg >> 8) << 16;
        const int nm = (m & 1) + ((m >> 1) & 1);
        const long long i0 = it.start / R;
        unsigned int c = 0;
        for (int i = lane; i < it.len / R; i += 32) {
            const int b = (I16 ? (int)((const uint16_t*)t_col)[i0 + i] : ((const int32_t*)t_col)[i0 + i]) + (I16 ? add : 0);
            c += live[b] ? 1u : 0u;
        }
        tot += (unsigned long long)c * R * nm;
    }
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_down_sync(0xffffffffu, tot, o);
    if (lane == 0 && tot) atomicAdd(out, tot);
}

// Second stage of a transposed pass: one thread per spot adds the spot's partial sums in slot order (ascending
// structure, then ascending position in the run) and runs the epilogue: gradient store (a3), update + clamp (a9), or
// fp32 output.  Spots without entries keep g / output 0 (set at creation / by the caller); their x is still clamped.
template <int EPI>
__global__ void __launch_bounds__(256)
k_combine(long long S, const long long* __restrict__ item_ptr, const double* __restrict__ partial,
          double* __restrict__ g_out, double* __restrict__ gpart, double* __restrict__ x, const DevState* __restrict__ st,
          float* __restrict__ f_out) {
    pdl_wait();
    pdl_trigger();
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (EPI == TEPI_GRAD) {   // also the CTA's share of |g|^2 (fixed order), summed by k_select
        __shared__ double sm[8];
        double tot = 0.0;
        if (j < S) {
            const long long ib = item_ptr[j], ie = item_ptr[j + 1];
            for (long long i = ib; i < ie; ++i) tot += partial[i];
            if (ie > ib) g_out[j] = tot;
        }
        const double q = block_sum(tot * tot, sm);
        if (threadIdx.x == 0) gpart[blockIdx.x] = q;
        return;
    }
    if (j >= S) return;
    const long long ib = item_ptr[j], ie = item_ptr[j + 1];
    double tot = 0.0;
    for (long long i = ib; i < ie; ++i) tot += partial[i];
    if (EPI == TEPI_UPDATE) {                              // every spot is clamped, also one no labelled row touches (R6)
        const double v = ie > ib ? x[j] - st->relax * tot : x[j];   // x <- x' - lambda eta^k * sum w^ (r/|a|^2) a
        x[j] = v < 0.0 ? 0.0 : v;                          // clamp
    } else if (ie > ib) f_out[j] = (float)tot;
}

}  // namespace fredopt
