// fredopt_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded fp64 CPU restatement of the hot path of FREDopt's plan
// optimisation, written from the paper (/root/reference/PAPER.md, arxiv 2509.20012) and the
// readings recorded in DESIGN.md ("Readings of the paper", R0..R22 = SURVEY.md sec. 8c A0..A22).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may use
// it.  It shares no code with the CUDA path (paper_2509_20012_b200/csrc) and neither includes the
// other.
//
// What it computes, step by step in the paper's order and notation:
//   * AMSrelaxDLET (Fig. 2) in its SIMULTANEOUS (Cimmino) form (reading R1): every
//     residual is taken at the same fluence x and one summed, weighted, relaxed step is applied, then
//     the clamp fluence_j < 0 -> 0;
//   * SuperiorDLET (Fig. 3): before each AMS step, `reductionsN` perturbations
//     x' = x - beta * grad_cost(x), beta = beta0 * a^s, accepted only if cost(x') < cost(x);
//   * cost chi^2(x) of Eq. (2) and its gradient;
//   * LETd = l / d voxel-wise (Eq. (1) with the dose as denominator);
//   * the OAR LETd limit linearised as <L_i - LETmax*D_i, x> <= 0, the proximity function and the
//     violation count (not in the paper: BASELINE.json north_star; reading R18).
//
// Everything is double; the fp32 inputs are widened once.  Rows are visited in index order; the
// back-projection is an ordered scatter-add through the forward CSR (no transposed copy).  There is
// no blocking, fusion or reordering.
//
// Parity pins: tests/test_oracle_pins.py checks this file against dense brute force, closed forms
// and invariants (SURVEY.md sec. 8c pins 1-12).  The paper prints no worked numbers of an iteration
// and never states lambda, alpha, eta, reductionsN or the matrix sizes, so parity with the PAPER'S OWN
// RUNS is unpinned; the algorithmic content is pinned by those mathematical checks.

// Timing build: the same source compiled with -fopenmp (oracle.py build(omp=True)) runs the row loops of the simultaneous form
// on all host cores -- rows in static contiguous chunks, back-projections into per-thread private S-vectors that are added
// in thread order (SURVEY.md sec. 8d "Oracle timing").  Without -fopenmp the pragmas vanish and every loop is the plain
// index-order loop; with one thread the two builds give the same bits (tests/test_oracle_pins.py::test_openmp_*).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// Row loop of a pass: body(i, acc, t) handles row i, adding its S-vector contribution into acc (null if the pass has none) and
// its scalar contributions into slot t of the caller's per-slot accumulators.  Plain build: one pass in index order, acc = out,
// t = 0.  OpenMP build: static contiguous chunks of rows, per-thread private vectors added to `out` in thread order.
inline int row_slots() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
template <class Body>
void for_rows(int64_t V, int64_t S, std::vector<double>* out, Body body) {
    if (out) out->assign(S, 0.0);
#ifdef _OPENMP
    const int nt = omp_get_max_threads();
    if (nt > 1) {
        std::vector<std::vector<double>> priv(out ? nt : 0);
#pragma omp parallel num_threads(nt)
        {
            const int t = omp_get_thread_num();
            std::vector<double>* acc = nullptr;
            if (out) { priv[t].assign(S, 0.0); acc = &priv[t]; }
#pragma omp for schedule(static)
            for (int64_t i = 0; i < V; ++i) body(i, acc, t);
        }
        if (out)
            for (int t = 0; t < nt; ++t)
                for (int64_t j = 0; j < S; ++j) (*out)[j] += priv[t][j];
        return;
    }
#endif
    for (int64_t i = 0; i < V; ++i) body(i, out, 0);
}

struct Csr {
    int64_t n_rows = 0, n_cols = 0;
    std::vector<int64_t> ptr;
    std::vector<int32_t> col;
    std::vector<double> val;   // widened once from fp32
};

struct Bounds {   // all widened from the fp32 bit patterns the caller passed; NaN = absent
    double weight, dose_lo, dose_hi, dl_lo, dl_hi, letd_max, dose_ref, dl_ref;
};

inline bool present(double v) { return !std::isnan(v); }

// fields of the per-voxel bound arrays (bounds "defined for each point in the image space"; Eq. (2),
// per-voxel Dref_i, cDLref_i)
enum { VB_DOSE_LO = 0, VB_DOSE_HI, VB_DL_LO, VB_DL_HI, VB_LETD_MAX, VB_DOSE_REF, VB_DL_REF, VB_N };

struct Plan {
    Csr D, L;
    std::vector<int32_t> label;        // per voxel; 0 = unconstrained
    std::vector<Bounds> bounds;        // index s-1 for label s
    std::vector<double> vb[VB_N];      // optional per-voxel values (empty = none; NaN = the structure's scalar)
    std::vector<double> nD, nL, nT;    // squared norms of D_i, L_i, L_i - letd_max*D_i  (per voxel)
    std::vector<double> what;          // normalised weight per structure (index s-1)
    double W = 0.0;
    int64_t n_sets = 0, n_zero_norm_sets = 0;
    std::vector<double> x;             // fluence
    // state of Fig. 3
    int64_t k = 0, s = 0, trials = 0;
    bool started = false;              // beta0, a latched (first superiorized call after create / reset)
    double latched_beta0 = 0.0, latched_a = 0.0;
    double beta_next = 0.0, eta_pow = 1.0, last_beta = 0.0;
    // options
    double eta = 1.0;
    int64_t reductionsN = 1, max_trials = 200;
    bool accept_check = true;
    bool normalize_grad = false;       // reading R9 option: step along g / |g|_2
    bool one_sided_cost = false;       // reading R11 option: OAR term (cDL - cDLref)_+^2
    bool block_sequential = false;     // reading R23: Fig. 2's loop nest, sequential over (kind, ROI) blocks
    double sweep_prox = 0.0;           // statistics of the last block-sequential sweep (at visit time)
    int64_t sweep_viol = 0;
};

// Bounds of voxel i (structure s): the structure's scalars, each replaced by the voxel's own value where a per-voxel array
// holds one.  Which constraint kinds and cost terms a voxel has is decided by its structure (has_dose_slab(bounds[s-1]), ...).
inline Bounds voxel_bounds(const Plan& P, int64_t i, int32_t s) {
    Bounds b = P.bounds[s - 1];
    double* f[VB_N] = {&b.dose_lo, &b.dose_hi, &b.dl_lo, &b.dl_hi, &b.letd_max, &b.dose_ref, &b.dl_ref};
    for (int k = 0; k < VB_N; ++k)
        if (!P.vb[k].empty() && !std::isnan(P.vb[k][i])) *f[k] = P.vb[k][i];
    return b;
}

// <A_i, x>
inline double row_dot(const Csr& A, int64_t i, const std::vector<double>& x) {
    double acc = 0.0;
    for (int64_t p = A.ptr[i]; p < A.ptr[i + 1]; ++p) acc += A.val[p] * x[A.col[p]];
    return acc;
}

bool has_dose_slab(const Bounds& b) { return present(b.dose_lo) || present(b.dose_hi); }
bool has_dl_slab(const Bounds& b) { return present(b.dl_lo) || present(b.dl_hi); }
bool has_letd(const Bounds& b) { return present(b.letd_max); }

// Signed residual of a hyperslab lo <= val <= hi (reading R5: one set per (row, quantity); R2: sign):
// upper violations positive, lower violations negative, 0 inside.
inline double slab_residual(double val, double lo, double hi) {
    if (present(hi) && val > hi) return val - hi;
    if (present(lo) && val < lo) return val - lo;
    return 0.0;
}

// <L_i - letd_max * D_i, x> over the union pattern of rows i of L and D (merge of two sorted rows).
double letd_row_dot(const Plan& P, int64_t i, double letd_max, const std::vector<double>& x, double* norm2) {
    const Csr &D = P.D, &L = P.L;
    int64_t p = D.ptr[i], pe = D.ptr[i + 1], q = L.ptr[i], qe = L.ptr[i + 1];
    double acc = 0.0, n2 = 0.0;
    while (p < pe || q < qe) {
        int32_t cd = p < pe ? D.col[p] : INT32_MAX, cl = q < qe ? L.col[q] : INT32_MAX;
        double a;
        int32_t c;
        if (cd == cl) { a = L.val[q] - letd_max * D.val[p]; c = cd; ++p; ++q; }
        else if (cd < cl) { a = -letd_max * D.val[p]; c = cd; ++p; }
        else { a = L.val[q]; c = cl; ++q; }
        acc += a * x[c];
        n2 += a * a;
    }
    if (norm2) *norm2 = n2;
    return acc;
}

void setup(Plan& P) {
    const int64_t V = P.D.n_rows;
    P.nD.assign(V, 0.0); P.nL.assign(V, 0.0); P.nT.assign(V, 0.0);
    std::vector<int64_t> part(P.bounds.size(), 0);   // participating sets per structure
    std::vector<double> zero(P.D.n_cols, 0.0);
    P.n_sets = 0; P.n_zero_norm_sets = 0;
    for (int64_t i = 0; i < V; ++i) {
        int32_t s = P.label[i];
        if (s == 0) continue;
        const Bounds& b = P.bounds[s - 1];
        double n = 0.0;
        for (int64_t p = P.D.ptr[i]; p < P.D.ptr[i + 1]; ++p) n += P.D.val[p] * P.D.val[p];
        P.nD[i] = n;
        n = 0.0;
        for (int64_t p = P.L.ptr[i]; p < P.L.ptr[i + 1]; ++p) n += P.L.val[p] * P.L.val[p];
        P.nL[i] = n;
        if (has_letd(b)) { letd_row_dot(P, i, voxel_bounds(P, i, s).letd_max, zero, &n); P.nT[i] = n; }
        if (has_dose_slab(b)) { ++P.n_sets; if (P.nD[i] > 0) ++part[s - 1]; else ++P.n_zero_norm_sets; }
        if (has_dl_slab(b))   { ++P.n_sets; if (P.nL[i] > 0) ++part[s - 1]; else ++P.n_zero_norm_sets; }
        if (has_letd(b))      { ++P.n_sets; if (P.nT[i] > 0) ++part[s - 1]; else ++P.n_zero_norm_sets; }
    }
    // reading R3: w^_s = w_s / W,  W = sum over participating sets of w_{s(k)} (grouped by structure, s ascending)
    P.W = 0.0;
    for (size_t s = 0; s < P.bounds.size(); ++s) P.W += P.bounds[s].weight * (double)part[s];
    P.what.assign(P.bounds.size(), 0.0);
    for (size_t s = 0; s < P.bounds.size(); ++s) P.what[s] = P.W > 0 ? P.bounds[s].weight / P.W : 0.0;
}

// chi^2(x), Eq. (2): sum_i w^_i (Dref_i - D(x)_i)^2 + sum_i w^_i (cDLref_i - cDL(x)_i)^2
double cost(const Plan& P, const std::vector<double>& x) {
    double phi = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : phi)
    for (int64_t i = 0; i < P.D.n_rows; ++i) {
        int32_t s = P.label[i];
        if (s == 0) continue;
        const Bounds& sb = P.bounds[s - 1];                         // the structure decides which terms exist ...
        const Bounds b = voxel_bounds(P, i, s);                      // ... the voxel may carry its own reference values
        if (present(sb.dose_ref)) { double e = b.dose_ref - row_dot(P.D, i, x); phi += P.what[s - 1] * e * e; }
        if (present(sb.dl_ref))   { double e = b.dl_ref - row_dot(P.L, i, x);
                                   if (!(P.one_sided_cost && e > 0.0)) phi += P.what[s - 1] * e * e; }   // one-sided: only cDL above cDLref
    }
    return phi;
}

// grad chi^2(x) = 2 [ sum_i w^_i (D(x)_i - Dref_i) D_i + sum_i w^_i (cDL(x)_i - cDLref_i) L_i ]
void grad_cost(const Plan& P, const std::vector<double>& x, std::vector<double>& g) {
    for_rows(P.D.n_rows, P.D.n_cols, &g, [&](int64_t i, std::vector<double>* gp, int) {
        std::vector<double>& g = *gp;
        int32_t s = P.label[i];
        if (s == 0) return;
        const Bounds& sb = P.bounds[s - 1];
        const Bounds b = voxel_bounds(P, i, s);
        if (present(sb.dose_ref)) {
            double c = 2.0 * P.what[s - 1] * (row_dot(P.D, i, x) - b.dose_ref);
            for (int64_t p = P.D.ptr[i]; p < P.D.ptr[i + 1]; ++p) g[P.D.col[p]] += c * P.D.val[p];
        }
        if (present(sb.dl_ref)) {
            double c = 2.0 * P.what[s - 1] * (row_dot(P.L, i, x) - b.dl_ref);
            if (P.one_sided_cost && c < 0.0) c = 0.0;
            for (int64_t p = P.L.ptr[i]; p < P.L.ptr[i + 1]; ++p) g[P.L.col[p]] += c * P.L.val[p];
        }
    });
}

// One pass over all declared sets at x.  If `step` is non-null it receives
//   sum_{k in P} w^_k (r_k / n_k) a_k      (the summed Fig. 2 step fractions)
// prox = 1/2 sum_{k in P} w^_k r_k^2 / n_k ;  n_viol = #{declared sets with r_k != 0}.
void constraint_pass(const Plan& P, const std::vector<double>& x, std::vector<double>* step,
                     double* prox, int64_t* n_viol) {
    std::vector<double> prs(row_slots(), 0.0);      // one slot in the plain build: the sums run in index order
    std::vector<int64_t> nvs(row_slots(), 0);
    for_rows(P.D.n_rows, P.D.n_cols, step, [&](int64_t i, std::vector<double>* step, int t) {
        double& pr = prs[t];
        int64_t& nv = nvs[t];
        int32_t s = P.label[i];
        if (s == 0) return;
        const Bounds& sb = P.bounds[s - 1];
        const Bounds b = voxel_bounds(P, i, s);
        const double w = P.what[s - 1];
        if (has_dose_slab(sb)) {                                  // dose block of Fig. 2 (R4)
            double r = slab_residual(row_dot(P.D, i, x), b.dose_lo, b.dose_hi);
            if (r != 0.0) ++nv;
            if (P.nD[i] > 0 && r != 0.0) {
                pr += 0.5 * w * r * r / P.nD[i];
                if (step) { double c = w * r / P.nD[i];
                    for (int64_t p = P.D.ptr[i]; p < P.D.ptr[i + 1]; ++p) (*step)[P.D.col[p]] += c * P.D.val[p]; }
            }
        }
        if (has_dl_slab(sb)) {                                    // cDLET block of Fig. 2
            double r = slab_residual(row_dot(P.L, i, x), b.dl_lo, b.dl_hi);
            if (r != 0.0) ++nv;
            if (P.nL[i] > 0 && r != 0.0) {
                pr += 0.5 * w * r * r / P.nL[i];
                if (step) { double c = w * r / P.nL[i];
                    for (int64_t p = P.L.ptr[i]; p < P.L.ptr[i + 1]; ++p) (*step)[P.L.col[p]] += c * P.L.val[p]; }
            }
        }
        if (has_letd(sb)) {                                       // <L_i - LETmax D_i, x> <= 0 (north_star)
            double val = letd_row_dot(P, i, b.letd_max, x, nullptr);
            double r = val > 0.0 ? val : 0.0;
            if (r != 0.0) ++nv;
            if (P.nT[i] > 0 && r != 0.0) {
                pr += 0.5 * w * r * r / P.nT[i];
                if (step) { double c = w * r / P.nT[i];
                    for (int64_t p = P.L.ptr[i]; p < P.L.ptr[i + 1]; ++p) (*step)[P.L.col[p]] += c * P.L.val[p];
                    for (int64_t p = P.D.ptr[i]; p < P.D.ptr[i + 1]; ++p) (*step)[P.D.col[p]] -= c * b.letd_max * P.D.val[p]; }
            }
        }
    });
    double pr = 0.0;
    int64_t nv = 0;
    for (size_t t = 0; t < prs.size(); ++t) { pr += prs[t]; nv += nvs[t]; }
    if (prox) *prox = pr;
    if (n_viol) *n_viol = nv;
}

// Block-sequential AMS sweep (reading R23): the loop nest of Fig. 2 -- first the dose kind over all
// ROIs in label order, then the cDLET kind, then the LETd rows of north_star -- taken block by block: SEQUENTIAL over
// the (kind, ROI) blocks, SIMULTANEOUS inside a block.  For block b = (kind, ROI s) with participating rows
// P_b = {i in s : |a_i|^2 > 0}, m = |P_b|:
//     x <- x - relax * min(w_s, 1) * (1/m) * sum_{i in P_b} (r_i / |a_i|^2) a_i,     every r_i taken at the x the block starts from
// (the per-row step fractions of Fig. 2 averaged over the block; min(w_s, 1) is the structure's priority as a relaxation
// factor).  The clamp of PAPER.md:149-154 follows the last block.  Statistics: sets found violated when their
// block is visited, and 1/2 sum w^_s r_i^2/|a_i|^2 over them (global w^ of R3).
void block_sweep(Plan& P, double relax) {
    const int64_t V = P.D.n_rows, S = P.D.n_cols;
    std::vector<double>& x = P.x;
    std::vector<double> step(S);
    P.sweep_prox = 0.0; P.sweep_viol = 0;
    for (int kind = 0; kind < 3; ++kind)
        for (size_t s = 1; s <= P.bounds.size(); ++s) {
            const Bounds& b = P.bounds[s - 1];
            if (kind == 0 ? !has_dose_slab(b) : kind == 1 ? !has_dl_slab(b) : !has_letd(b)) continue;
            std::fill(step.begin(), step.end(), 0.0);
            int64_t m = 0;
            for (int64_t i = 0; i < V; ++i) {
                if (P.label[i] != (int32_t)s) continue;
                const Bounds vbn = voxel_bounds(P, i, (int32_t)s);
                double r, n;
                if (kind == 0) { r = slab_residual(row_dot(P.D, i, x), vbn.dose_lo, vbn.dose_hi); n = P.nD[i]; }
                else if (kind == 1) { r = slab_residual(row_dot(P.L, i, x), vbn.dl_lo, vbn.dl_hi); n = P.nL[i]; }
                else { double val = letd_row_dot(P, i, vbn.letd_max, x, nullptr); r = val > 0.0 ? val : 0.0; n = P.nT[i]; }
                if (r != 0.0) ++P.sweep_viol;
                if (!(n > 0.0)) continue;
                ++m;
                if (r == 0.0) continue;
                P.sweep_prox += 0.5 * P.what[s - 1] * r * r / n;
                const double c = r / n;
                if (kind == 0) for (int64_t p = P.D.ptr[i]; p < P.D.ptr[i + 1]; ++p) step[P.D.col[p]] += c * P.D.val[p];
                else if (kind == 1) for (int64_t p = P.L.ptr[i]; p < P.L.ptr[i + 1]; ++p) step[P.L.col[p]] += c * P.L.val[p];
                else {
                    for (int64_t p = P.L.ptr[i]; p < P.L.ptr[i + 1]; ++p) step[P.L.col[p]] += c * P.L.val[p];
                    for (int64_t p = P.D.ptr[i]; p < P.D.ptr[i + 1]; ++p) step[P.D.col[p]] -= c * vbn.letd_max * P.D.val[p];
                }
            }
            if (m == 0) continue;
            const double f = relax * (b.weight < 1.0 ? b.weight : 1.0) / (double)m;
            for (int64_t j = 0; j < S; ++j) x[j] -= f * step[j];
        }
    for (int64_t j = 0; j < S; ++j) if (x[j] < 0.0) x[j] = 0.0;
}

void fill_csr(Csr& A, int64_t V, int64_t S, const int64_t* ptr, const int32_t* col, const float* val) {
    A.n_rows = V; A.n_cols = S;
    A.ptr.assign(ptr, ptr + V + 1);
    int64_t nnz = ptr[V];
    A.col.assign(col, col + nnz);
    A.val.resize(nnz);
    for (int64_t p = 0; p < nnz; ++p) A.val[p] = (double)val[p];
}

}  // namespace

extern "C" {

void* oracle_create(int64_t V, int64_t S, const int64_t* ptrD, const int32_t* colD, const float* valD,
                    const int64_t* ptrL, const int32_t* colL, const float* valL, const int32_t* labels,
                    const float* bounds /* n_struct x 8: weight, dose_lo, dose_hi, dl_lo, dl_hi, letd_max, dose_ref, dl_ref */,
                    int32_t n_struct) {
    Plan* P = new Plan();
    fill_csr(P->D, V, S, ptrD, colD, valD);
    fill_csr(P->L, V, S, ptrL, colL, valL);
    P->label.assign(labels, labels + V);
    for (int32_t s = 0; s < n_struct; ++s) {
        const float* b = bounds + 8 * s;
        P->bounds.push_back(Bounds{(double)b[0], (double)b[1], (double)b[2], (double)b[3], (double)b[4],
                                   (double)b[5], (double)b[6], (double)b[7]});
    }
    P->x.assign(S, 0.0);
    setup(*P);
    return P;
}

void oracle_destroy(void* h) { delete (Plan*)h; }

// threads the row loops run on (1 in the plain build)
int32_t oracle_threads(void) { return (int32_t)row_slots(); }
void oracle_set_threads(int32_t n) {
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

void oracle_set_x(void* h, const float* x) { Plan* P = (Plan*)h; for (size_t j = 0; j < P->x.size(); ++j) P->x[j] = (double)x[j]; }
void oracle_set_x64(void* h, const double* x) { Plan* P = (Plan*)h; P->x.assign(x, x + P->x.size()); }
void oracle_get_x(void* h, double* x) { Plan* P = (Plan*)h; std::memcpy(x, P->x.data(), P->x.size() * sizeof(double)); }

// keys: 0 eta, 1 reductionsN, 2 accept_check, 3 max_trials, 4 reset (k, s, beta), 7 block-sequential AMS (R23), 8 normalised gradient (R9), 9 one-sided cDL cost (R11)
void oracle_set_option(void* h, int32_t key, double v) {
    Plan* P = (Plan*)h;
    switch (key) {
        case 0: P->eta = v; break;
        case 1: P->reductionsN = (int64_t)v; break;
        case 2: P->accept_check = v != 0.0; break;
        case 3: P->max_trials = (int64_t)v; break;
        case 4: P->k = 0; P->s = 0; P->trials = 0; P->started = false; P->eta_pow = 1.0; P->last_beta = 0.0; break;
        case 7: P->block_sequential = v != 0.0; break;
        case 8: P->normalize_grad = v != 0.0; break;
        case 9: P->one_sided_cost = v != 0.0; break;
        default: break;
    }
}

// Per-voxel values of one bound field (V floats, NaN = the structure's scalar; NULL removes the array).  A value applies where
// the voxel's structure declares that kind of constraint / cost term.  Norms and w^ are set up again (the LETd rows
// L_i - LETmax_i D_i change with LETmax_i).  Returns 0, or -1 (nothing changed) if a value is infinite or lo > hi on a voxel.
int32_t oracle_set_voxel_bounds(void* h, int32_t field, const float* values) {
    Plan* P = (Plan*)h;
    if (field < 0 || field >= VB_N) return -1;
    const int64_t V = P->D.n_rows;
    std::vector<double> old = P->vb[field];
    if (!values) P->vb[field].clear();
    else {
        P->vb[field].resize(V);
        for (int64_t i = 0; i < V; ++i) P->vb[field][i] = (double)values[i];
    }
    bool ok = true;
    for (int64_t i = 0; i < V && ok; ++i) {
        if (values && std::isinf(values[i])) ok = false;
        if (P->label[i] == 0) continue;
        const Bounds b = voxel_bounds(*P, i, P->label[i]);
        if (b.dose_lo > b.dose_hi || b.dl_lo > b.dl_hi) ok = false;
    }
    if (!ok) { P->vb[field] = old; return -1; }
    setup(*P);
    return 0;
}

// d = D x, l = L x over ALL rows; LETd_i = l_i / d_i where d_i > 0, else 0 (Eq. (1); R15)
void oracle_dose_let(void* h, const double* xin, double* dose, double* l_out, double* letd) {
    Plan* P = (Plan*)h;
    std::vector<double> x = xin ? std::vector<double>(xin, xin + P->x.size()) : P->x;
    for (int64_t i = 0; i < P->D.n_rows; ++i) {
        double d = row_dot(P->D, i, x), l = row_dot(P->L, i, x);
        if (dose) dose[i] = d;
        if (l_out) l_out[i] = l;
        if (letd) letd[i] = d > 0.0 ? l / d : 0.0;
    }
}

// Same as oracle_dose_let but only for the listed rows (full-size sampled parity).
void oracle_dose_let_rows(void* h, const double* xin, const int64_t* rows, int64_t n, double* dose, double* l_out, double* letd) {
    Plan* P = (Plan*)h;
    std::vector<double> x = xin ? std::vector<double>(xin, xin + P->x.size()) : P->x;
    for (int64_t t = 0; t < n; ++t) {
        int64_t i = rows[t];
        double d = row_dot(P->D, i, x), l = row_dot(P->L, i, x);
        dose[t] = d; l_out[t] = l; letd[t] = d > 0.0 ? l / d : 0.0;
    }
}

// out_j = sum_i D_ij u_i + L_ij v_i over all rows (active_only: rows with label != 0), ordered scatter-add.
// out_abs_j = sum_i |D_ij u_i| + |L_ij v_i|  (the scale the per-element tolerance refers to).
void oracle_transpose(void* h, const double* u, const double* v, int32_t active_only, double* out, double* out_abs) {
    Plan* P = (Plan*)h;
    const int64_t S = P->D.n_cols;
    for (int64_t j = 0; j < S; ++j) { out[j] = 0.0; if (out_abs) out_abs[j] = 0.0; }
    for (int64_t i = 0; i < P->D.n_rows; ++i) {
        if (active_only && P->label[i] == 0) continue;
        if (u) for (int64_t p = P->D.ptr[i]; p < P->D.ptr[i + 1]; ++p) {
            double t = P->D.val[p] * u[i]; out[P->D.col[p]] += t; if (out_abs) out_abs[P->D.col[p]] += std::fabs(t); }
        if (v) for (int64_t p = P->L.ptr[i]; p < P->L.ptr[i + 1]; ++p) {
            double t = P->L.val[p] * v[i]; out[P->L.col[p]] += t; if (out_abs) out_abs[P->L.col[p]] += std::fabs(t); }
    }
}

double oracle_cost(void* h, const double* xin) {
    Plan* P = (Plan*)h;
    std::vector<double> x = xin ? std::vector<double>(xin, xin + P->x.size()) : P->x;
    return cost(*P, x);
}

void oracle_grad(void* h, const double* xin, double* g) {
    Plan* P = (Plan*)h;
    std::vector<double> x = xin ? std::vector<double>(xin, xin + P->x.size()) : P->x, gv;
    grad_cost(*P, x, gv);
    std::memcpy(g, gv.data(), gv.size() * sizeof(double));
}

void oracle_proximity(void* h, const double* xin, double* prox, int64_t* n_viol) {
    Plan* P = (Plan*)h;
    std::vector<double> x = xin ? std::vector<double>(xin, xin + P->x.size()) : P->x;
    constraint_pass(*P, x, nullptr, prox, n_viol);
}

// SuperiorDLET (Fig. 3) around the simultaneous AMSrelaxDLET step (Fig. 2).
// lambda, beta0, a arrive as the fp32 bit patterns the caller passes to the C-ABI and are widened here.
// The step-size sequence beta_s = beta0 a^s (R8) belongs to the plan: beta0 and a are latched by the first call with
// beta0 > 0 and n_iter > 0 after create / reset; a later call with beta0 > 0 must pass the same pair (else -1 and nothing
// is done); calls with beta0 == 0 (pure feasibility-seeking) neither latch nor consume the sequence.  Returns 0 / -1.
int32_t oracle_iterate(void* h, int32_t n_iter, float lambda_f, float beta0_f, float a_f) {
    Plan* P = (Plan*)h;
    const double lambda = (double)lambda_f, beta0 = (double)beta0_f, a = (double)a_f;
    const int64_t S = P->D.n_cols;
    if (beta0 != 0.0 && n_iter > 0) {
        if (!P->started) { P->beta_next = beta0; P->latched_beta0 = beta0; P->latched_a = a; P->started = true; }   // beta_0 = beta0
        else if (beta0 != P->latched_beta0 || a != P->latched_a) return -1;
    }
    std::vector<double> g, xn(S), step;
    for (int32_t it = 0; it < n_iter; ++it) {
        // ---- perturbation phase; skipped entirely when beta0 == 0 (pure AMS)
        if (beta0 != 0.0) {
            for (int64_t t = 0; t < P->reductionsN; ++t) {
                const double phi0 = cost(*P, P->x);
                grad_cost(*P, P->x, g);
                bool zero = true;
                for (int64_t j = 0; j < S; ++j) if (g[j] != 0.0) { zero = false; break; }
                if (zero) break;                                              // R10: nothing to reduce
                if (P->normalize_grad) {                                      // R9 option: unit direction g / |g|_2
                    double n2 = 0.0;
                    for (int64_t j = 0; j < S; ++j) n2 += g[j] * g[j];
                    const double inv = 1.0 / std::sqrt(n2);
                    for (int64_t j = 0; j < S; ++j) g[j] *= inv;
                }
                for (int64_t trial = 0; trial < P->max_trials; ++trial) {     // `while loop do`; R10 cap
                    const double beta = P->beta_next;                        // s = s + 1; beta = alpha^s (R8: beta0 * a^s)
                    P->beta_next *= a; ++P->s; ++P->trials;
                    for (int64_t j = 0; j < S; ++j) xn[j] = P->x[j] - beta * g[j];
                    if (!P->accept_check || cost(*P, xn) < phi0) {            // strict decrease
                        P->x = xn; P->last_beta = beta; break;
                    }
                }
            }
        }
        // ---- feasibility-seeking step with w_k = eta^k w, simultaneous form (R1)
        const double relax = lambda * P->eta_pow;
        if (P->block_sequential) block_sweep(*P, relax);                       // R23: Fig. 2's own loop nest, block by block
        else {
            constraint_pass(*P, P->x, &step, nullptr, nullptr);
            for (int64_t j = 0; j < S; ++j) {
                double v = P->x[j] - relax * step[j];
                P->x[j] = v < 0.0 ? 0.0 : v;                                   // clamp (R6)
            }
        }
        P->eta_pow *= P->eta;
        ++P->k;
    }
    return 0;
}

// out: k, s, trials, n_sets, n_zero_norm_sets ; dout: last_beta, W, beta_next
void oracle_stats(void* h, int64_t* out, double* dout) {
    Plan* P = (Plan*)h;
    out[0] = P->k; out[1] = P->s; out[2] = P->trials; out[3] = P->n_sets; out[4] = P->n_zero_norm_sets;
    dout[0] = P->last_beta; dout[1] = P->W; dout[2] = P->beta_next;
}

// The state of Fig. 3 carried from call to call (checkpoint / resume): iout = k, s, trials, latched; dout = beta_next, eta_pow,
// last_beta, latched beta0, latched a.
void oracle_get_state(void* h, int64_t* iout, double* dout) {
    Plan* P = (Plan*)h;
    iout[0] = P->k; iout[1] = P->s; iout[2] = P->trials; iout[3] = P->started ? 1 : 0;
    dout[0] = P->beta_next; dout[1] = P->eta_pow; dout[2] = P->last_beta; dout[3] = P->latched_beta0; dout[4] = P->latched_a;
}
void oracle_set_state(void* h, const int64_t* iin, const double* din) {
    Plan* P = (Plan*)h;
    P->k = iin[0]; P->s = iin[1]; P->trials = iin[2]; P->started = iin[3] != 0;
    P->beta_next = din[0]; P->eta_pow = din[1]; P->last_beta = din[2]; P->latched_beta0 = din[3]; P->latched_a = din[4];
}

void oracle_sweep_stats(void* h, double* prox, int64_t* n_viol) {
    Plan* P = (Plan*)h;
    *prox = P->sweep_prox; *n_viol = P->sweep_viol;
}

// ---- evaluation quantities of PAPER.md:110 (DVH, LVH, cDLVH, cDL30) and Table 1 -- SURVEY sec. 8f-3.
// Values of one voxel quantity over the voxels of structure `label`, in voxel order:
// quantity 0: dose d_i = <D_i, x>; 1: cDL l_i = <L_i, x>; 2: LETd l_i / d_i (0 where d_i = 0, R15).
static std::vector<double> structure_values(const Plan& P, const std::vector<double>& x, int quantity, int label) {
    std::vector<double> v;
    for (int64_t i = 0; i < P.D.n_rows; ++i) {
        if (P.label[i] != label) continue;
        const double d = row_dot(P.D, i, x), l = row_dot(P.L, i, x);
        v.push_back(quantity == 0 ? d : quantity == 1 ? l : (d > 0.0 ? l / d : 0.0));
    }
    return v;
}

// min, mean, max over the structure's voxels (Table 1's columns) and the voxel count; all 0 for an empty structure
void oracle_structure_stats(void* h, const double* xin, int32_t quantity, int32_t label, double* out3, int64_t* n) {
    Plan* P = (Plan*)h;
    std::vector<double> x = xin ? std::vector<double>(xin, xin + P->x.size()) : P->x;
    std::vector<double> v = structure_values(*P, x, quantity, label);
    *n = (int64_t)v.size();
    out3[0] = out3[1] = out3[2] = 0.0;
    if (v.empty()) return;
    double mn = v[0], mx = v[0], sum = 0.0;
    for (double t : v) { mn = t < mn ? t : mn; mx = t > mx ? t : mx; sum += t; }
    out3[0] = mn; out3[1] = sum / (double)v.size(); out3[2] = mx;
}

// cumulative volume histogram: hist[b] = fraction of the structure's voxels with value >= b * vmax / n_bins
void oracle_volume_histogram(void* h, const double* xin, int32_t quantity, int32_t label, int32_t n_bins, double vmax, double* hist) {
    Plan* P = (Plan*)h;
    std::vector<double> x = xin ? std::vector<double>(xin, xin + P->x.size()) : P->x;
    std::vector<double> v = structure_values(*P, x, quantity, label);
    for (int32_t b = 0; b < n_bins; ++b) {
        int64_t c = 0;
        const double edge = (double)b * vmax / (double)n_bins;
        for (double t : v) if (t >= edge) ++c;
        hist[b] = v.empty() ? 0.0 : (double)c / (double)v.size();
    }
}

// "the value received by `fraction` of the structure volume" (cDL30: fraction 0.3): the smallest of the
// ceil(fraction * n) largest values, i.e. the largest t such that at least fraction * n voxels have a value >= t
double oracle_percentile_value(void* h, const double* xin, int32_t quantity, int32_t label, double fraction) {
    Plan* P = (Plan*)h;
    std::vector<double> x = xin ? std::vector<double>(xin, xin + P->x.size()) : P->x;
    std::vector<double> v = structure_values(*P, x, quantity, label);
    if (v.empty()) return 0.0;
    std::sort(v.begin(), v.end(), [](double a, double b) { return a > b; });
    int64_t k = (int64_t)std::ceil(fraction * (double)v.size());
    if (k < 1) k = 1;
    if (k > (int64_t)v.size()) k = (int64_t)v.size();
    return v[k - 1];
}

void oracle_norms(void* h, double* nD, double* nL, double* nT) {
    Plan* P = (Plan*)h;
    std::memcpy(nD, P->nD.data(), P->nD.size() * sizeof(double));
    std::memcpy(nL, P->nL.data(), P->nL.size() * sizeof(double));
    std::memcpy(nT, P->nT.data(), P->nT.size() * sizeof(double));
}

void oracle_what(void* h, double* what) { Plan* P = (Plan*)h; std::memcpy(what, P->what.data(), P->what.size() * sizeof(double)); }

// Fully sequential Fig. 2 sweep exactly as the listing reads (in-place updates voxel by voxel, dose block then
// cDLET block, then the LETd rows, then the clamp) with per-row relaxation lambda * weight_s (un-normalised):
// tiny-case sanity reference only (SURVEY pin 12); NOT the method under test.
void oracle_sequential_sweep(void* h, float lambda_f) {
    Plan* P = (Plan*)h;
    const double lambda = (double)lambda_f;
    std::vector<double>& x = P->x;
    for (int pass = 0; pass < 3; ++pass)
        for (int64_t i = 0; i < P->D.n_rows; ++i) {
            int32_t s = P->label[i];
            if (s == 0) continue;
            const Bounds& sb = P->bounds[s - 1];
            const Bounds b = voxel_bounds(*P, i, s);
            const double w = b.weight < 1.0 ? b.weight : 1.0;
            if (pass == 0 && has_dose_slab(sb) && P->nD[i] > 0) {
                double r = slab_residual(row_dot(P->D, i, x), b.dose_lo, b.dose_hi);
                if (r != 0.0) { double c = lambda * w * r / P->nD[i];
                    for (int64_t p = P->D.ptr[i]; p < P->D.ptr[i + 1]; ++p) x[P->D.col[p]] -= c * P->D.val[p]; }
            }
            if (pass == 1 && has_dl_slab(sb) && P->nL[i] > 0) {
                double r = slab_residual(row_dot(P->L, i, x), b.dl_lo, b.dl_hi);
                if (r != 0.0) { double c = lambda * w * r / P->nL[i];
                    for (int64_t p = P->L.ptr[i]; p < P->L.ptr[i + 1]; ++p) x[P->L.col[p]] -= c * P->L.val[p]; }
            }
            if (pass == 2 && has_letd(sb) && P->nT[i] > 0) {
                double val = letd_row_dot(*P, i, b.letd_max, x, nullptr);
                if (val > 0.0) { double c = lambda * w * val / P->nT[i];
                    for (int64_t p = P->L.ptr[i]; p < P->L.ptr[i + 1]; ++p) x[P->L.col[p]] -= c * P->L.val[p];
                    for (int64_t p = P->D.ptr[i]; p < P->D.ptr[i + 1]; ++p) x[P->D.col[p]] += c * b.letd_max * P->D.val[p]; }
            }
        }
    for (size_t j = 0; j < x.size(); ++j) if (x[j] < 0.0) x[j] = 0.0;
}

}  // extern "C"
