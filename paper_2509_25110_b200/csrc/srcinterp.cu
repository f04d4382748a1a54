// srcinterp.cu -- InterpolateSources (SourceToTransfers "begins by calling
// IntegrationVars_init ... and InterpolateSources to prepare the source data"): the
// sources leave the perturbation evolution on a coarse wavenumber grid and are brought onto the k grid of
// the line-of-sight integration.  The paper does not say how; reading R26: for every tau,
// independently, the NATURAL cubic spline in k through (kc_i, S(kc_i, tau)), evaluated at the plan's k.
//
//   h_{i-1}/6 M_{i-1} + (h_{i-1}+h_i)/3 M_i + h_i/6 M_{i+1} = (y_{i+1}-y_i)/h_i - (y_i-y_{i-1})/h_{i-1},
//   M_0 = M_{n-1} = 0,  s(k) = A y_i + B y_{i+1} + ((A^3-A) M_i + (B^3-B) M_{i+1}) h_i^2/6.
//
// The matrix depends on the coarse grid only: its LU factors, and per fine k its interval and the four
// weights (A, B, (A^3-A) h^2/6, (B^3-B) h^2/6), are tables of the handle, built once on the host.
// Arrays are [k][tau] with tau fastest, so thread <-> tau makes every access of both kernels coalesced:
//   solve:  M = A^-1 d with the banded inverse of the spline matrix as a dense contraction on the FP64 tensor
//           cores (srcinterp_mma_kernel); grids the band does not serve: one thread per (series, tau) walks the
//           coarse grid down and up (srcinterp_solve_kernel: two dependent FMA chains of n_kc steps);
//           second derivatives M to scratch;
//   eval:   one thread per (series, k, two tau): four coarse values (L2-resident) -> one fine value, the
//           HBM-bound part (8 n_k n_tau bytes written per series).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdint>
#include <new>
#include <vector>

#include "los_internal.cuh"

// -DGCAMB_DEBUG (GCAMB_DEBUG=1 python -m paper_2509_25110_b200.build --force): device asserts on the indices
#ifdef GCAMB_DEBUG
#include <cassert>
#define GCAMB_ASSERT(c) assert(c)
#else
#define GCAMB_ASSERT(c) ((void)0)
#endif

struct gcamb_los_srcinterp {
    int32_t n_kc, n_k, n_tau, device;
    double *d_h;          // [n_kc]   h_i = kc_{i+1} - kc_i (last entry unused)
    double *d_ih;         // [n_kc]   1 / h_i (an fp64 division is ~40 dependent instructions: none in the sweeps)
    double *d_mult;       // [n_kc]   forward-elimination multipliers
    double *d_inv_diag;   // [n_kc]   reciprocals of the eliminated diagonal
    int32_t *d_seg;       // [n_k]    coarse interval of every fine k
    double4 *d_wgt;       // [n_k]    (A, B, (A^3-A) h^2/6, (B^3-B) h^2/6)
    // banded form of the solve (see srcinterp_mma_kernel); n_iblk = 0: the sequential sweeps are used
    double *d_blk_val;    // A fragments of the banded inverse: per block of 8 rows and k-step, 32 lane-ordered values
    int32_t *d_blk_off, *d_blk_jlo, *d_blk_ks;   // [n_iblk] offset into d_blk_val, first column, k-steps of 4 columns
    int32_t *d_grp_j0, *d_grp_kw;                // [n_grp] first row and number of rows of d a thread block needs
    int32_t n_iblk, n_grp, kw_max, band_max;     // band_max: columns of the widest row
};

// Scratch of gcamb_los_interp_sources_noalloc: the second derivatives of the splines, [n_series][n_kc][n_tau]
// doubles, at most NOALLOC_SCRATCH_DOUBLES of them (8 MiB).  A file-scope device array: every GPU that loads the
// library holds it until the process exits, and every call on a device shares it.  In HOST code the name is a
// host-side stand-in, not a device address: the kernels get the address cudaGetSymbolAddress returns (below).
constexpr size_t NOALLOC_SCRATCH_DOUBLES = (size_t)1 << 20;
static __device__ __align__(256) double g_noalloc_scratch[NOALLOC_SCRATCH_DOUBLES];

namespace gcamb {

namespace {

// SMEM: the thread's column of the series is first copied into shared memory ([n_kc][blockDim], conflict-free)
// with independent, unrolled loads (a dependent sweep through global memory pays a DRAM round trip per step:
// measured 252 us for 300 knots), swept there in place, and written back; the three coefficient tables sit
// in shared memory too.  Without SMEM (coarse grids too long for shared memory) the sweeps go through M in
// global memory.
template <bool SMEM>
__global__ void __launch_bounds__(128) srcinterp_solve_kernel(const double *__restrict__ S_c, double *__restrict__ M,
                                                              const double *__restrict__ h, const double *__restrict__ ih,
                                                              const double *__restrict__ mult,
                                                              const double *__restrict__ inv_diag, int n_kc, int n_tau)
{
    extern __shared__ double sm_r[];
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = t < n_tau;
    const int rs = blockDim.x;
    const size_t base = (size_t)blockIdx.y * n_kc * n_tau + (active ? t : 0);
    const double *y = S_c + base;
    double *m = M + base;
    if (SMEM) {
        double *r_s = sm_r + threadIdx.x;            // [i * blockDim]
        double *tab = sm_r + (size_t)n_kc * rs;      // 1/h | mult | inv_diag h/6
        for (int i = threadIdx.x; i < n_kc; i += rs) {
            tab[i] = ih[i]; tab[n_kc + i] = mult[i]; tab[2 * n_kc + i] = inv_diag[i]; tab[3 * n_kc + i] = h[i] * (1.0 / 6.0);
        }
        if (active) {
#pragma unroll 16
            for (int i = 0; i < n_kc; ++i) r_s[i * rs] = y[(size_t)i * n_tau];
        }
        __syncthreads();
        if (!active) return;
        if (n_kc >= 3) {
            double y0 = r_s[0], y1 = r_s[rs], r = 0.0;
#pragma unroll 8
            for (int i = 1; i < n_kc - 1; ++i) {
                const double y2 = r_s[(i + 1) * rs];
                const double d = fma(y2 - y1, tab[i], -((y1 - y0) * tab[i - 1]));
                r = fma(-tab[n_kc + i], r, d);          // mult_1 = 0
                r_s[i * rs] = r;
                y0 = y1;
                y1 = y2;
            }
            double next = 0.0;
#pragma unroll 8
            for (int i = n_kc - 2; i >= 1; --i) {
                next = fma(-tab[3 * n_kc + i], next, r_s[i * rs]) * tab[2 * n_kc + i];
                r_s[i * rs] = next;
            }
        }
        r_s[0] = 0.0;
        r_s[(n_kc - 1) * rs] = 0.0;
#pragma unroll 16
        for (int i = 0; i < n_kc; ++i) m[(size_t)i * n_tau] = r_s[i * rs];
        return;
    }
    if (!active) return;
    m[0] = 0.0;
    m[(size_t)(n_kc - 1) * n_tau] = 0.0;
    if (n_kc < 3) return;
    // forward: r_i = d_i - mult_i r_{i-1},  d_i = (y_{i+1}-y_i)/h_i - (y_i-y_{i-1})/h_{i-1}
    double y0 = y[0], y1 = y[n_tau], r = 0.0;
    for (int i = 1; i < n_kc - 1; ++i) {
        const double y2 = y[(size_t)(i + 1) * n_tau];
        const double d = fma(y2 - y1, ih[i], -((y1 - y0) * ih[i - 1]));
        r = fma(-mult[i], r, d);
        m[(size_t)i * n_tau] = r;
        y0 = y1;
        y1 = y2;
    }
    // back substitution: M_i = (r_i - h_i/6 M_{i+1}) / diag_i
    double next = 0.0;
    for (int i = n_kc - 2; i >= 1; --i) {
        next = fma(-h[i] * (1.0 / 6.0), next, m[(size_t)i * n_tau]) * inv_diag[i];
        m[(size_t)i * n_tau] = next;
    }
}

// The spline matrix is tridiagonal and diagonally dominant by a factor 2 in every row, whatever the grid, so the
// entries of its inverse fall off at least like 2^-|i-j| (Neumann series; 0.27^|i-j| on a nearly uniform grid):
// M_i = sum_j (A^-1)_ij d_j needs ~30 columns either side of the diagonal, and every (i, tau) is independent of
// every other, where the two sweeps of the Thomas algorithm are 2400 dependent chains of 300 steps (73 us, bound
// by the latency of the chain).  The rows of A^-1 are built on the host at creation and cut where the dropped
// entries, weighted with the largest right-hand side they can meet and the largest weight the evaluation gives
// M_i, sum to less than 1e-18 max|S| (a bound, not an estimate).
// With the band, M[8 rows x tau] = A^-1[8 x K] . d[K x tau] (K ~ 72) is a dense contraction: it runs on the FP64
// tensor cores (mma.sync.m8n8k4.f64), ONE operand load per 256 multiply-adds.  (The same dot products on the plain
// FP64 pipe, one thread per tau: 75 us, every FMA waits for its two operand loads: long_scoreboard 16 per issue.)
// Block = MM_WARPS warps x MM_TAU tau: the right-hand sides d_j of the rows the block's bands reach are formed
// from the coarse sources (coalesced along tau) into shared memory; warp w then takes the 8 rows of "i-block"
// 4 group + w: A fragments straight from the host-packed table (lane-ordered, zero outside a row's band: one
// coalesced 256-byte load per k-step, shared through L1 by the warps of all tau), B fragments from shared memory.
constexpr int MM_WARPS = 4;
constexpr int MM_TAU = 32;     // tau per block = 4 MMA column tiles per warp
constexpr int MM_DS = 36;      // row stride of d in shared memory: 4 rows x 8 tau of a B fragment hit distinct banks
constexpr int MM_KW_MAX = 200; // rows of d a block may need (57.6 KB)

__device__ __forceinline__ void dmma_884(double (&d)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(32 * MM_WARPS) srcinterp_mma_kernel(const double *__restrict__ S_c, double *__restrict__ M,
                                                                      const double *__restrict__ ih, const double *__restrict__ blk_val,
                                                                      const int32_t *__restrict__ blk_off, const int32_t *__restrict__ blk_jlo,
                                                                      const int32_t *__restrict__ blk_ks, const int32_t *__restrict__ grp_j0,
                                                                      const int32_t *__restrict__ grp_kw, int n_kc, int n_tau, int n_iblk)
{
    extern __shared__ double dsm[];                 // [Kw][MM_DS]
    // the evaluation kernel behind this one is launched with programmatic stream serialization: its thread blocks
    // may become resident as soon as every block of this grid has started, and wait (griddepcontrol.wait) for
    // this grid to complete before they read M
    asm volatile("griddepcontrol.launch_dependents;");
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tau0 = blockIdx.x * MM_TAU, grp = blockIdx.y;
    const int wj0 = grp_j0[grp], Kw = grp_kw[grp];
    const size_t base = (size_t)blockIdx.z * n_kc * n_tau;
    // right-hand sides d_j = (y_{j+1} - y_j) / h_j - (y_j - y_{j-1}) / h_{j-1}, j = wj0 .. wj0 + Kw - 1; zero outside
    // the interior rows and past the end of the tau grid (the A fragments are zero there, but 0 x NaN is not)
    {
        const int t = tau0 + lane;
        const bool tv = t < n_tau;
        const double *y = S_c + base + (tv ? t : 0);
        auto row = [&](int q) { return (tv && q >= 0 && q < n_kc) ? y[(size_t)q * n_tau] : 0.0; };
        const int per = (Kw + MM_WARPS - 1) / MM_WARPS;             // a warp takes consecutive rows: one new load per row
        const int r0 = warp * per, r1 = min(Kw, r0 + per);
        if (r0 < r1) {
            double y0 = row(wj0 + r0 - 1), y1 = row(wj0 + r0);
#pragma unroll 8
            for (int r = r0; r < r1; ++r) {
                const int j = wj0 + r;
                const double y2 = row(j + 1);
                GCAMB_ASSERT(r >= 0 && r < Kw && Kw <= MM_KW_MAX && j >= 0 && j <= n_kc + 4 * MM_WARPS);
                double d = 0.0;
                if (tv && j >= 1 && j <= n_kc - 2) d = fma(y2 - y1, __ldg(ih + j), -((y1 - y0) * __ldg(ih + j - 1)));
                dsm[r * MM_DS + lane] = d;
                y0 = y1;
                y1 = y2;
            }
        }
    }
    __syncthreads();
    const int b = grp * MM_WARPS + warp;            // this warp's rows: 8 b .. 8 b + 7
    if (b >= n_iblk) return;
    const int ks = blk_ks[b], fr = lane >> 2, fc = lane & 3;
    const double *av = blk_val + blk_off[b] + lane;
    const double *dp = dsm + (blk_jlo[b] - wj0 + fc) * MM_DS + fr;
    GCAMB_ASSERT(blk_jlo[b] >= wj0 && blk_jlo[b] - wj0 + 4 * ks <= Kw && blk_off[b] >= 0);   // every B fragment row lies in the block's window
    double D[MM_TAU / 8][2];
#pragma unroll
    for (int nt = 0; nt < MM_TAU / 8; ++nt) D[nt][0] = D[nt][1] = 0.0;
#pragma unroll 4
    for (int s = 0; s < ks; ++s) {
        const double a = __ldg(av + 32 * s);        // A[row fr][column 4 s + fc]
#pragma unroll
        for (int nt = 0; nt < MM_TAU / 8; ++nt) dmma_884(D[nt], a, dp[4 * s * MM_DS + 8 * nt]);   // B[k fc][tau 8 nt + fr]
    }
    // D fragment: row fr, tau 8 nt + 2 fc, + 1.  Rows 0 and n_kc - 1 carry zero coefficients: M_0 = M_{n-1} = 0.
    const int row = 8 * b + fr;
    if (row < n_kc) {
        double *m = M + base + (size_t)row * n_tau;
#pragma unroll
        for (int nt = 0; nt < MM_TAU / 8; ++nt) {
            const int t = tau0 + 8 * nt + 2 * fc;
            GCAMB_ASSERT(row >= 0 && row < n_kc && t >= 0);
            if (t < n_tau) m[t] = D[nt][0];
            if (t + 1 < n_tau) m[t + 1] = D[nt][1];
        }
    }
}

constexpr int EVAL_ROWS = 8;   // fine k rows per CTA (one row per CTA: 30000 one-shot CTAs, 33 us for 58 MB)

// s(k_j, tau) = A y_s + B y_{s+1} + C M_s + D M_{s+1}.  VEC = 2: two tau per thread through 16-byte loads and stores
// (n_tau even, buffers 16-byte aligned); the scalar form of the kernel issued 70 instructions per warp and row and
// was bound by instruction issue (66 % of the issue slots), not by memory.  Both forms do the same operations in
// the same order on every element.
__device__ __forceinline__ double spline_value(const double4 &w, double ya, double yb, double ma, double mb)
{
    return fma(w.x, ya, w.y * yb) + fma(w.z, ma, w.w * mb);
}

template <int VEC>
__global__ void __launch_bounds__(256) srcinterp_eval_kernel(const double *__restrict__ S_c, const double *__restrict__ M,
                                                             const int32_t *__restrict__ seg, const double4 *__restrict__ wgt,
                                                             double *__restrict__ S_f, int n_kc, int n_k, int n_tau)
{
    const size_t cbase = (size_t)blockIdx.z * n_kc * n_tau;
    const int j0 = blockIdx.y * EVAL_ROWS, j_end = min(n_k, j0 + EVAL_ROWS);
    // launched with programmatic stream serialization: the block becomes resident while the solve kernel drains and
    // waits here until M is complete and visible
    asm volatile("griddepcontrol.wait;" ::: "memory");
    for (int t = (blockIdx.x * blockDim.x + threadIdx.x) * VEC; t < n_tau; t += gridDim.x * blockDim.x * VEC) {
#pragma unroll 4
        for (int j = j0; j < j_end; ++j) {
            const int sg = __ldg(seg + j);           // the same for the whole block: broadcast loads
            const double4 w = wgt[j];
            const size_t c = cbase + (size_t)sg * n_tau + t, f = ((size_t)blockIdx.z * n_k + j) * n_tau + t;
            GCAMB_ASSERT(sg >= 0 && sg + 1 < n_kc && t + VEC <= n_tau && j < n_k);
            if (VEC == 2) {
                const double2 ya = *reinterpret_cast<const double2 *>(S_c + c), yb = *reinterpret_cast<const double2 *>(S_c + c + n_tau);
                const double2 ma = *reinterpret_cast<const double2 *>(M + c), mb = *reinterpret_cast<const double2 *>(M + c + n_tau);
                *reinterpret_cast<double2 *>(S_f + f) = make_double2(spline_value(w, ya.x, yb.x, ma.x, mb.x),
                                                                     spline_value(w, ya.y, yb.y, ma.y, mb.y));
            } else {
                S_f[f] = spline_value(w, S_c[c], S_c[c + n_tau], M[c], M[c + n_tau]);
            }
        }
    }
}

}  // namespace
}  // namespace gcamb

using namespace gcamb;

extern "C" {

gcamb_status gcamb_los_srcinterp_create(gcamb_los_srcinterp **out, const gcamb_los_plan *plan,
                                        const double *k_coarse, int32_t n_kc, void *cuda_stream)
{
    if (out) *out = nullptr;
    if (!out || !plan || !k_coarse) { set_error("null argument"); return GCAMB_EINVAL; }
    const double *k_fine = plan->h_k;
    if (n_kc < 2) { set_error("need at least two coarse wavenumbers"); return GCAMB_EINVAL; }
    for (int i = 0; i < n_kc; ++i) {
        if (!std::isfinite(k_coarse[i]) || !(k_coarse[i] > 0.0)) { set_error("k_coarse[%d] must be finite and > 0", i); return GCAMB_EGRID; }
        if (i && !(k_coarse[i] > k_coarse[i - 1])) { set_error("k_coarse not strictly increasing at %d", i); return GCAMB_EGRID; }
    }
    const int n_k = plan->n_k;
    for (int j = 0; j < n_k; ++j)
        if (!(k_fine[j] >= k_coarse[0] && k_fine[j] <= k_coarse[n_kc - 1])) {
            set_error("k[%d] lies outside the coarse grid: the spline does not extrapolate", j);
            return GCAMB_EGRID;
        }
    int dev = -1;
    GCAMB_CUDA(cudaGetDevice(&dev));
    if (dev != plan->device) { set_error("plan belongs to device %d but device %d is current", plan->device, dev); return GCAMB_EINVAL; }

    std::vector<double> h(n_kc, 0.0), mult(n_kc, 0.0), inv_diag(n_kc, 0.0), diag(n_kc, 0.0);
    for (int i = 0; i + 1 < n_kc; ++i) h[i] = k_coarse[i + 1] - k_coarse[i];
    std::vector<double> ih(n_kc, 0.0);
    for (int i = 0; i + 1 < n_kc; ++i) ih[i] = 1.0 / h[i];
    for (int i = 1; i < n_kc - 1; ++i) diag[i] = (h[i - 1] + h[i]) / 3.0;
    for (int i = 2; i < n_kc - 1; ++i) {
        const double sub = h[i - 1] / 6.0;
        mult[i] = sub / diag[i - 1];
        diag[i] -= mult[i] * sub;
    }
    for (int i = 1; i < n_kc - 1; ++i) inv_diag[i] = 1.0 / diag[i];
    // Banded inverse (srcinterp_mma_kernel).  Row i of A^-1 = the solution of A x = e_i (A is symmetric) through the
    // factors above, in long double; it is cut on both sides where the dropped entries can add at most 0.5e-18 max|S|
    // to an interpolated value: |d_j| <= 2 max|S| (1/h_j + 1/h_{j-1}), and M_i enters a value with a weight of at most
    // 0.385 max(h_{i-1}, h_i)^2 / 6.  Grids whose rows stay wide (average above BAND_MAX_AVG columns: spacings that
    // jump by orders of magnitude) and very long grids keep the sequential sweeps.
    constexpr int BAND_MAX_KC = 4096, BAND_MAX_AVG = 100;
    std::vector<double> ainv;
    std::vector<double> blk_val;
    std::vector<int32_t> a_off(n_kc, 0), a_lo(n_kc, 0), a_cnt(n_kc, 0), blk_off, blk_jlo, blk_ks, grp_j0, grp_kw;
    int kw_max = 0, band_max = 0;
    bool band_ok = false;
    if (n_kc >= 3 && n_kc <= BAND_MAX_KC) {
        std::vector<long double> r(n_kc), x(n_kc);
        std::vector<double> g(n_kc, 0.0);
        for (int j = 1; j < n_kc - 1; ++j) g[j] = 2.0 * (ih[j] + ih[j - 1]);
        bool ok = true;
        for (int i = 1; i < n_kc - 1 && ok; ++i) {
            for (int j = 1; j < n_kc - 1; ++j) r[j] = 0.0L;
            r[i] = 1.0L;
            for (int j = i + 1; j < n_kc - 1; ++j) r[j] = -(long double)mult[j] * r[j - 1];
            long double next = 0.0L;
            for (int j = n_kc - 2; j >= 1; --j) { next = (r[j] - (long double)h[j] / 6.0L * next) / (long double)diag[j]; x[j] = next; }
            const double hm = std::max(h[i - 1], h[i]);
            const long double budget = 0.5e-18L / (0.385L * hm * hm / 6.0L);
            int lo = 1, hi = n_kc - 2;
            long double tail = 0.0L;
            while (lo < i && tail + fabsl(x[lo]) * g[lo] <= budget) { tail += fabsl(x[lo]) * g[lo]; ++lo; }
            tail = 0.0L;
            while (hi > i && tail + fabsl(x[hi]) * g[hi] <= budget) { tail += fabsl(x[hi]) * g[hi]; --hi; }
            a_off[i] = (int32_t)ainv.size(); a_lo[i] = lo; a_cnt[i] = hi - lo + 1;
            band_max = std::max(band_max, hi - lo + 1);
            for (int j = lo; j <= hi; ++j) ainv.push_back((double)x[j]);
            if (ainv.size() > (size_t)BAND_MAX_AVG * (size_t)n_kc) ok = false;
        }
        if (ok) {
            // A fragments: block b = rows 8 b .. 8 b + 7, columns jlo_b + 4 s + c; value of lane 4 r + c, zero outside the row's band
            const int n_iblk = (n_kc + 7) / 8;
            for (int bk = 0; bk < n_iblk; ++bk) {
                int jlo = n_kc, jhi = -1;
                for (int i = std::max(1, 8 * bk); i < std::min(n_kc - 1, 8 * bk + 8); ++i) {
                    jlo = std::min(jlo, a_lo[i]);
                    jhi = std::max(jhi, a_lo[i] + a_cnt[i] - 1);
                }
                const int ks = jhi >= jlo ? (jhi - jlo + 1 + 3) / 4 : 0;
                blk_off.push_back((int32_t)blk_val.size()); blk_jlo.push_back(ks ? jlo : 1); blk_ks.push_back(ks);
                for (int st = 0; st < ks; ++st)
                    for (int ln = 0; ln < 32; ++ln) {
                        const int i = 8 * bk + (ln >> 2), jcol = jlo + 4 * st + (ln & 3);
                        double v = 0.0;
                        if (i >= 1 && i <= n_kc - 2 && jcol >= a_lo[i] && jcol < a_lo[i] + a_cnt[i]) v = ainv[a_off[i] + (jcol - a_lo[i])];
                        blk_val.push_back(v);
                    }
            }
            const int n_grp = (n_iblk + MM_WARPS - 1) / MM_WARPS;
            for (int gq = 0; gq < n_grp; ++gq) {
                int j0 = n_kc, j1 = 0;
                for (int bk = gq * MM_WARPS; bk < std::min(n_iblk, (gq + 1) * MM_WARPS); ++bk)
                    if (blk_ks[bk]) { j0 = std::min(j0, blk_jlo[bk]); j1 = std::max(j1, blk_jlo[bk] + 4 * blk_ks[bk]); }
                grp_j0.push_back(j1 > j0 ? j0 : 1);
                grp_kw.push_back(j1 > j0 ? j1 - j0 : 0);
                kw_max = std::max(kw_max, grp_kw.back());
            }
            band_ok = kw_max <= MM_KW_MAX;
        }
    }
    std::vector<int32_t> seg(n_k);
    std::vector<double4> wgt(n_k);
    for (int j = 0; j < n_k; ++j) {
        int s = (int)(std::upper_bound(k_coarse, k_coarse + n_kc, k_fine[j]) - k_coarse) - 1;
        s = std::max(0, std::min(s, n_kc - 2));
        if (s > 0 && k_fine[j] == k_coarse[s]) --s;       // a knot belongs to the interval on its left, like the search "k > kc[s+1]"
        const double hh = h[s];
        const double A = (k_coarse[s + 1] - k_fine[j]) / hh, B = (k_fine[j] - k_coarse[s]) / hh;
        seg[j] = s;
        wgt[j] = make_double4(A, B, (A * A * A - A) * (hh * hh) / 6.0, (B * B * B - B) * (hh * hh) / 6.0);
    }
    gcamb_los_srcinterp *si = new (std::nothrow) gcamb_los_srcinterp();
    if (!si) { set_error("out of host memory"); return GCAMB_EALLOC; }
    *si = gcamb_los_srcinterp{};
    si->n_kc = n_kc; si->n_k = n_k; si->n_tau = plan->n_tau; si->device = dev;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaMalloc(&si->d_h, sizeof(double) * n_kc);
    if (e == cudaSuccess) e = cudaMalloc(&si->d_ih, sizeof(double) * n_kc);
    if (e == cudaSuccess) e = cudaMalloc(&si->d_mult, sizeof(double) * n_kc);
    if (e == cudaSuccess) e = cudaMalloc(&si->d_inv_diag, sizeof(double) * n_kc);
    if (e == cudaSuccess) e = cudaMalloc(&si->d_seg, sizeof(int32_t) * n_k);
    if (e == cudaSuccess) e = cudaMalloc(&si->d_wgt, sizeof(double4) * n_k);
    if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_h, h.data(), sizeof(double) * n_kc, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_ih, ih.data(), sizeof(double) * n_kc, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_mult, mult.data(), sizeof(double) * n_kc, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_inv_diag, inv_diag.data(), sizeof(double) * n_kc, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_seg, seg.data(), sizeof(int32_t) * n_k, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_wgt, wgt.data(), sizeof(double4) * n_k, cudaMemcpyHostToDevice, s);
    if (band_ok) {
        const size_t nb = blk_off.size(), ng = grp_j0.size();
        si->n_iblk = (int32_t)nb; si->n_grp = (int32_t)ng; si->kw_max = kw_max; si->band_max = band_max;
        if (e == cudaSuccess) e = cudaMalloc(&si->d_blk_val, sizeof(double) * std::max<size_t>(blk_val.size(), 1));
        if (e == cudaSuccess) e = cudaMalloc(&si->d_blk_off, sizeof(int32_t) * nb);
        if (e == cudaSuccess) e = cudaMalloc(&si->d_blk_jlo, sizeof(int32_t) * nb);
        if (e == cudaSuccess) e = cudaMalloc(&si->d_blk_ks, sizeof(int32_t) * nb);
        if (e == cudaSuccess) e = cudaMalloc(&si->d_grp_j0, sizeof(int32_t) * ng);
        if (e == cudaSuccess) e = cudaMalloc(&si->d_grp_kw, sizeof(int32_t) * ng);
        if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_blk_val, blk_val.data(), sizeof(double) * blk_val.size(), cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_blk_off, blk_off.data(), sizeof(int32_t) * nb, cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_blk_jlo, blk_jlo.data(), sizeof(int32_t) * nb, cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_blk_ks, blk_ks.data(), sizeof(int32_t) * nb, cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_grp_j0, grp_j0.data(), sizeof(int32_t) * ng, cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(si->d_grp_kw, grp_kw.data(), sizeof(int32_t) * ng, cudaMemcpyHostToDevice, s);
        // opt in to the shared memory of the widest block here, once, so that a call only launches
        if (e == cudaSuccess && sizeof(double) * (size_t)kw_max * MM_DS > 48 * 1024)
            e = cudaFuncSetAttribute(srcinterp_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(double) * MM_KW_MAX * MM_DS));
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);   // the vectors die with this scope
    if (e != cudaSuccess) {
        gcamb_status st = cuda_fail(e, "gcamb_los_srcinterp_create");
        gcamb_los_srcinterp_destroy(si);
        return st;
    }
    *out = si;
    return GCAMB_OK;
}

gcamb_status gcamb_los_srcinterp_destroy(gcamb_los_srcinterp *si)
{
    if (!si) return GCAMB_OK;
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e == cudaSuccess && cur != si->device) e = cudaSetDevice(si->device);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    cudaFree(si->d_h); cudaFree(si->d_ih); cudaFree(si->d_mult); cudaFree(si->d_inv_diag); cudaFree(si->d_seg); cudaFree(si->d_wgt);
    cudaFree(si->d_blk_val); cudaFree(si->d_blk_off); cudaFree(si->d_blk_jlo); cudaFree(si->d_blk_ks); cudaFree(si->d_grp_j0); cudaFree(si->d_grp_kw);
    if (cur >= 0 && cur != si->device) cudaSetDevice(cur);
    delete si;
    if (e != cudaSuccess) return cuda_fail(e, "gcamb_los_srcinterp_destroy");
    return GCAMB_OK;
}

gcamb_status gcamb_los_srcinterp_info(const gcamb_los_srcinterp *si, int32_t *n_kc, int32_t *n_k, int32_t *n_tau,
                                      int32_t *band_columns)
{
    if (!si) { set_error("null handle"); return GCAMB_EINVAL; }
    if (n_kc) *n_kc = si->n_kc;
    if (n_k) *n_k = si->n_k;
    if (n_tau) *n_tau = si->n_tau;
    if (band_columns) *band_columns = si->n_iblk ? si->band_max : 0;
    return GCAMB_OK;
}

gcamb_status gcamb_los_interp_sources(const gcamb_los_srcinterp *si, int32_t n_series, const double *d_S_coarse,
                                      double *d_S_fine, double *d_work, void *cuda_stream)
{
    if (!si || !d_S_coarse || !d_S_fine || !d_work) { set_error("null handle or buffer"); return GCAMB_EINVAL; }
    if (n_series < 1 || n_series > 65535) { set_error("n_series must be in [1, 65535]"); return GCAMB_EINVAL; }
    if (si->n_k > 65535 * EVAL_ROWS) { set_error("n_k above 524280 not supported by the source interpolation"); return GCAMB_EINVAL; }
    int dev = -1;
    GCAMB_CUDA(cudaGetDevice(&dev));
    if (dev != si->device) { set_error("handle belongs to device %d but device %d is current", si->device, dev); return GCAMB_EINVAL; }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (si->n_iblk) {   // solve with the banded inverse on the FP64 tensor cores
        dim3 gb((unsigned)((si->n_tau + MM_TAU - 1) / MM_TAU), (unsigned)si->n_grp, (unsigned)n_series);
        srcinterp_mma_kernel<<<gb, 32 * MM_WARPS, sizeof(double) * (size_t)si->kw_max * MM_DS, s>>>(
            d_S_coarse, d_work, si->d_ih, si->d_blk_val, si->d_blk_off, si->d_blk_jlo, si->d_blk_ks, si->d_grp_j0, si->d_grp_kw,
            si->n_kc, si->n_tau, si->n_iblk);
        GCAMB_CUDA(cudaGetLastError());
    } else {
    // solve: 64 or 32 threads per block with the sweeps' intermediate in shared memory while it fits
    const size_t per_thread = sizeof(double) * (size_t)si->n_kc, tables = 4 * per_thread;
    const int threads = per_thread * 32 + tables <= 200 * 1024 ? 32 : 128;
    dim3 g1((unsigned)((si->n_tau + threads - 1) / threads), (unsigned)n_series);
    if (threads < 128) {
        const size_t smem = per_thread * threads + tables;
        if (smem > 48 * 1024)
            GCAMB_CUDA(cudaFuncSetAttribute(srcinterp_solve_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        srcinterp_solve_kernel<true><<<g1, threads, smem, s>>>(d_S_coarse, d_work, si->d_h, si->d_ih, si->d_mult, si->d_inv_diag, si->n_kc, si->n_tau);
    } else {
        srcinterp_solve_kernel<false><<<g1, threads, 0, s>>>(d_S_coarse, d_work, si->d_h, si->d_ih, si->d_mult, si->d_inv_diag, si->n_kc, si->n_tau);
    }
    GCAMB_CUDA(cudaGetLastError());
    }
    const bool vec2 = si->n_tau % 2 == 0 &&
                      ((reinterpret_cast<uintptr_t>(d_S_coarse) | reinterpret_cast<uintptr_t>(d_work) | reinterpret_cast<uintptr_t>(d_S_fine)) & 15) == 0;
    const int per_block = 256 * (vec2 ? 2 : 1);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)std::min((si->n_tau + per_block - 1) / per_block, 16), (unsigned)((si->n_k + EVAL_ROWS - 1) / EVAL_ROWS), (unsigned)n_series);
    cfg.blockDim = dim3(256);
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const double *c_Sc = d_S_coarse, *c_M = d_work;
    const int32_t *c_seg = si->d_seg;
    const double4 *c_wgt = si->d_wgt;
    GCAMB_CUDA(cudaLaunchKernelEx(&cfg, vec2 ? srcinterp_eval_kernel<2> : srcinterp_eval_kernel<1>, c_Sc, c_M, c_seg, c_wgt, d_S_fine,
                                  si->n_kc, si->n_k, si->n_tau));
    return GCAMB_OK;
}

// Device address of g_noalloc_scratch on the current device: looked up once per device (the first call on it),
// with that device current, and kept.
static gcamb_status noalloc_scratch_address(int dev, double **out)
{
    constexpr int MAX_DEV = 64;
    static std::atomic<double *> cache[MAX_DEV];
    double *ptr = (dev >= 0 && dev < MAX_DEV) ? cache[dev].load(std::memory_order_acquire) : nullptr;
    if (!ptr) {
        GCAMB_CUDA(cudaGetSymbolAddress((void **)&ptr, g_noalloc_scratch));   // `dev` is current: the caller checked
        if (!ptr) { set_error("cudaGetSymbolAddress returned a null address for the static scratch"); return GCAMB_ECUDA; }
        if (dev >= 0 && dev < MAX_DEV) cache[dev].store(ptr, std::memory_order_release);
    }
    *out = ptr;
    return GCAMB_OK;
}

gcamb_status gcamb_los_interp_sources_noalloc(const gcamb_los_srcinterp *si, int32_t n_series,
                                              const double *d_S_coarse, double *d_S_fine, void *cuda_stream)
{
    if (!si || !d_S_coarse || !d_S_fine) { set_error("null handle or buffer"); return GCAMB_EINVAL; }
    if (n_series < 1 || n_series > 65535) { set_error("n_series must be in [1, 65535]"); return GCAMB_EINVAL; }
    const unsigned long long need = (unsigned long long)n_series * (unsigned long long)si->n_kc * (unsigned long long)si->n_tau;
    if (need > NOALLOC_SCRATCH_DOUBLES) {
        set_error("gcamb_los_interp_sources_noalloc: n_series * n_kc * n_tau = %llu doubles exceeds the static scratch of "
                  "%llu doubles (8 MiB): use gcamb_los_interp_sources with caller-owned scratch",
                  need, (unsigned long long)NOALLOC_SCRATCH_DOUBLES);
        return GCAMB_EINVAL;
    }
    int dev = -1;
    GCAMB_CUDA(cudaGetDevice(&dev));
    if (dev != si->device) { set_error("handle belongs to device %d but device %d is current", si->device, dev); return GCAMB_EINVAL; }
    double *scratch = nullptr;
    if (gcamb_status st = noalloc_scratch_address(dev, &scratch)) return st;
    // Nothing in the scratch has to start at zero: the solve kernel writes every element [series][0 .. n_kc-1][tau]
    // that the evaluation kernel reads, in the same stream order, so what an earlier call left behind is never read.
    return gcamb_los_interp_sources(si, n_series, d_S_coarse, d_S_fine, scratch, cuda_stream);
}

}  // extern "C"
