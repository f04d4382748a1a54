// interp.cu -- spectra on every multipole from spectra on the plan's sparse l list
// (CAMB computes "a number of explicitly computed multipoles" set by
// l_sample_boost and gets the others by "spline interpolation", footnote 5 PAPER.md:127,
// PAPER.md:256; the paper defines neither the spline nor the interpolated quantity).
//
// Reading R25: natural cubic spline in l of y(l) = l (l+1) C_l^{XY}, knots = the l list,
// C_l = y(l) / (l (l+1)) afterwards.  Its second derivatives M_i solve the tridiagonal system
//     h_{i-1}/6 M_{i-1} + (h_{i-1}+h_i)/3 M_i + h_i/6 M_{i+1} = (y_{i+1}-y_i)/h_i - (y_i-y_{i-1})/h_{i-1},
//     h_i = l_{i+1} - l_i,   M_0 = M_{n-1} = 0,
// whose matrix depends on the l list only: its LU factors (Thomas algorithm) are plan tables, built
// once; for lists of up to 2048 knots so are the rows of its (banded) inverse, see cl_interp_band_kernel.
// A call does, per (cosmology, spectrum), one thread block (longer lists):
//     y_i, right-hand sides                      all threads
//     forward sweep, back substitution           one thread: two dependent FMA chains of n_l steps
//                                                (n_l ~ 100 for a CAMB-like list: ~1 us)
//     s(l) = A y_i + B y_{i+1} + ((A^3-A) M_i + (B^3-B) M_{i+1}) h_i^2/6 on every integer l,
//     A = (l_{i+1}-l)/h_i, B = (l-l_i)/h_i       all threads, coalesced stores
// Deterministic: no atomics, the order of every operation is fixed.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <vector>

#include "los_internal.cuh"

namespace gcamb {

namespace {

constexpr int INTERP_THREADS = 256;

__global__ void __launch_bounds__(INTERP_THREADS) cl_interp_kernel(const double *__restrict__ Cl_samp,
                                                                   double *__restrict__ Cl_all,
                                                                   const int32_t *__restrict__ l_list,
                                                                   const int32_t *__restrict__ seg_of_l,
                                                                   const double *__restrict__ sp_mult,
                                                                   const double *__restrict__ sp_inv_diag,
                                                                   int n_l, int n_all)
{
    extern __shared__ double sm[];
    double *y = sm, *M = sm + n_l;          // M holds the right-hand sides first, then the solution
    int *lk = reinterpret_cast<int *>(sm + 2 * (size_t)n_l);   // the knots: every later look-up stays in shared memory
    const size_t series = blockIdx.x;       // (cosmology, spectrum)
    const double *c = Cl_samp + series * n_l;
    for (int i = threadIdx.x; i < n_l; i += INTERP_THREADS) {
        const int li = l_list[i];
        const double l = (double)li;
        lk[i] = li;
        y[i] = l * (l + 1.0) * c[i];
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n_l; i += INTERP_THREADS) {
        double r = 0.0;
        if (i >= 1 && i < n_l - 1) {
            const double h0 = (double)(lk[i] - lk[i - 1]), h1 = (double)(lk[i + 1] - lk[i]);
            r = (y[i + 1] - y[i]) / h1 - (y[i] - y[i - 1]) / h0;
        }
        M[i] = r;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        // forward elimination with the plan's multipliers, then back substitution; the table loads do not
        // depend on the chains and are unrolled ahead of them (one L2 round trip per step otherwise: 23 us
        // for 101 knots)
#pragma unroll 8
        for (int i = 2; i < n_l - 1; ++i) M[i] = fma(-__ldg(sp_mult + i), M[i - 1], M[i]);
        double next = 0.0;                  // M_{n-1} = 0
#pragma unroll 8
        for (int i = n_l - 2; i >= 1; --i) {
            const double sup = (double)(lk[i + 1] - lk[i]) * (1.0 / 6.0);
            next = fma(-sup, next, M[i]) * __ldg(sp_inv_diag + i);
            M[i] = next;
        }
        M[0] = 0.0;
        M[n_l - 1] = 0.0;
    }
    __syncthreads();
    const int l0 = lk[0];
    double *out = Cl_all + series * n_all;
#pragma unroll 4
    for (int a = threadIdx.x; a < n_all; a += INTERP_THREADS) {
        const int l = l0 + a, s = __ldg(seg_of_l + a);
        const int la = lk[s], lb = lk[s + 1];
        const double h = (double)(lb - la);
        const double A = (double)(lb - l) / h, B = (double)(l - la) / h;
        const double sv = A * y[s] + B * y[s + 1] +
                          ((A * A * A - A) * M[s] + (B * B * B - B) * M[s + 1]) * (h * h) / 6.0;
        out[a] = sv / ((double)l * ((double)l + 1.0));
    }
}

// Lists of up to BAND_MAX_KNOTS knots (CAMB-like lists have ~100): the matrix is diagonally dominant by a factor 2
// in every row, so its inverse is banded to any wanted accuracy; the plan holds the rows of the inverse, cut where
// what is dropped stays below 1e-18 max|y| in a value of the spline (a bound), and the second derivatives are
// independent dot products, M_i = sum_j (A^-1)_ij r_j, one thread per knot, instead of two sweeps by one thread.
// With nothing sequential left the evaluation is spread over INTERP_CHUNK multipoles per thread block (every block
// repeats the small solve): 26.6 -> 8 us for 101 knots and 2499 multipoles.
constexpr int BAND_MAX_KNOTS = 2048;
constexpr int INTERP_CHUNK = 512;

__global__ void __launch_bounds__(INTERP_THREADS) cl_interp_band_kernel(const double *__restrict__ Cl_samp,
                                                                        double *__restrict__ Cl_all,
                                                                        const int32_t *__restrict__ l_list,
                                                                        const int32_t *__restrict__ seg_of_l,
                                                                        const double *__restrict__ ainv,
                                                                        const int32_t *__restrict__ a_off,
                                                                        const int32_t *__restrict__ a_lo,
                                                                        const int32_t *__restrict__ a_cnt,
                                                                        int n_l, int n_all)
{
    extern __shared__ double sm[];
    double *y = sm, *r = sm + n_l, *M = sm + 2 * (size_t)n_l;
    int *lk = reinterpret_cast<int *>(sm + 3 * (size_t)n_l);
    const size_t series = blockIdx.x;       // (cosmology, spectrum); blockIdx.y: chunk of multipoles
    const double *c = Cl_samp + series * n_l;
    // Everything the block reads from global memory whose address does not depend on other loads is requested here,
    // in one round trip (the tables are cold: a step streams hundreds of MB through the L2 between two calls): the
    // knots and samples, this thread's first row of the inverse, the knot intervals of its multipoles.
    constexpr int PER = INTERP_CHUNK / INTERP_THREADS;
    const int a_base = blockIdx.y * INTERP_CHUNK + threadIdx.x;
    int sg[PER];
#pragma unroll
    for (int u = 0; u < PER; ++u) sg[u] = a_base + u * INTERP_THREADS < n_all ? __ldg(seg_of_l + a_base + u * INTERP_THREADS) : 0;
    const int i_first = threadIdx.x;
    const bool interior = i_first >= 1 && i_first < n_l - 1;
    const int off1 = interior ? __ldg(a_off + i_first) : 0, lo1 = interior ? __ldg(a_lo + i_first) : 0, cnt1 = interior ? __ldg(a_cnt + i_first) : 0;
    for (int i = threadIdx.x; i < n_l; i += INTERP_THREADS) {
        const int li = l_list[i];
        const double l = (double)li;
        lk[i] = li;
        y[i] = l * (l + 1.0) * c[i];
    }
    // this thread's row of the inverse on its way into the L2 while the right-hand sides are formed
    for (int q = 0; q < cnt1; q += 16) asm volatile("prefetch.global.L2 [%0];" ::"l"(ainv + off1 + q));
    __syncthreads();
    for (int i = threadIdx.x; i < n_l; i += INTERP_THREADS) {
        double v = 0.0;
        if (i >= 1 && i < n_l - 1) {
            const double h0 = (double)(lk[i] - lk[i - 1]), h1 = (double)(lk[i + 1] - lk[i]);
            v = (y[i + 1] - y[i]) / h1 - (y[i] - y[i - 1]) / h0;
        }
        r[i] = v;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n_l; i += INTERP_THREADS) {
        double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;   // four chains, added in a fixed order
        if (i >= 1 && i < n_l - 1) {
            const bool first = i == i_first;
            const double *a = ainv + (first ? off1 : __ldg(a_off + i));
            const double *rr = r + (first ? lo1 : __ldg(a_lo + i));
            const int cnt = first ? cnt1 : __ldg(a_cnt + i);
            int q = 0;
#pragma unroll 2
            for (; q + 4 <= cnt; q += 4) {
                acc0 = fma(__ldg(a + q), rr[q], acc0);
                acc1 = fma(__ldg(a + q + 1), rr[q + 1], acc1);
                acc2 = fma(__ldg(a + q + 2), rr[q + 2], acc2);
                acc3 = fma(__ldg(a + q + 3), rr[q + 3], acc3);
            }
            for (; q < cnt; ++q) acc0 = fma(__ldg(a + q), rr[q], acc0);
        }
        M[i] = (acc0 + acc1) + (acc2 + acc3);           // M_0 = M_{n-1} = 0
    }
    __syncthreads();
    const int l0 = lk[0];
    double *out = Cl_all + series * n_all;
#pragma unroll
    for (int u = 0; u < PER; ++u) {
        const int a = a_base + u * INTERP_THREADS;
        if (a < n_all) {
            const int l = l0 + a, s = sg[u];
            const int la = lk[s], lb = lk[s + 1];
            const double h = (double)(lb - la);
            const double A = (double)(lb - l) / h, B = (double)(l - la) / h;
            const double sv = A * y[s] + B * y[s + 1] +
                              ((A * A * A - A) * M[s] + (B * B * B - B) * M[s + 1]) * (h * h) / 6.0;
            out[a] = sv / ((double)l * ((double)l + 1.0));
        }
    }
}

}  // namespace

// Plan tables of the spline (host, fp64; the matrix depends on the l list only).
gcamb_status interp_plan_tables(gcamb_los_plan *p, const int32_t *l_list, cudaStream_t stream)
{
    const int n = p->n_l_out;
    if (n < 2) return GCAMB_OK;             // a single multipole cannot be interpolated: the call reports it
    std::vector<double> mult(n, 0.0), inv_diag(n, 0.0), diag(n, 0.0);
    for (int i = 1; i < n - 1; ++i)
        diag[i] = ((double)(l_list[i] - l_list[i - 1]) + (double)(l_list[i + 1] - l_list[i])) / 3.0;
    for (int i = 2; i < n - 1; ++i) {       // sub-diagonal of row i = super-diagonal of row i-1 = h_{i-1}/6
        const double sub = (double)(l_list[i] - l_list[i - 1]) / 6.0;
        mult[i] = sub / diag[i - 1];
        diag[i] -= mult[i] * sub;
    }
    for (int i = 1; i < n - 1; ++i) inv_diag[i] = 1.0 / diag[i];
    const int n_all = l_list[n - 1] - l_list[0] + 1;   // tensor plans: l_max also counts l + 1
    std::vector<int32_t> seg(n_all);
    int s = 0;
    for (int a = 0; a < n_all; ++a) {
        const int l = l_list[0] + a;
        while (s < n - 2 && l > l_list[s + 1]) ++s;
        seg[a] = s;
    }
    GCAMB_CUDA(cudaMalloc(&p->d_sp_mult, sizeof(double) * n));
    GCAMB_CUDA(cudaMalloc(&p->d_sp_inv_diag, sizeof(double) * n));
    GCAMB_CUDA(cudaMalloc(&p->d_sp_seg, sizeof(int32_t) * n_all));
    GCAMB_CUDA(cudaMemcpyAsync(p->d_sp_mult, mult.data(), sizeof(double) * n, cudaMemcpyHostToDevice, stream));
    GCAMB_CUDA(cudaMemcpyAsync(p->d_sp_inv_diag, inv_diag.data(), sizeof(double) * n, cudaMemcpyHostToDevice, stream));
    GCAMB_CUDA(cudaMemcpyAsync(p->d_sp_seg, seg.data(), sizeof(int32_t) * n_all, cudaMemcpyHostToDevice, stream));
    // Banded inverse (cl_interp_band_kernel).  A symmetric tridiagonal, a_i on the diagonal, c_i = h_i/6 between rows
    // i and i+1; with the pivots d_i of the elimination from the top and delta_i of the elimination from the bottom,
    //   (A^-1)_ii = 1 / (d_i + delta_i - a_i),  (A^-1)_{i,j+1} = -(c_j / delta_{j+1}) (A^-1)_ij  (j >= i),
    //   (A^-1)_{i,j-1} = -(c_{j-1} / d_{j-1}) (A^-1)_ij  (j <= i).
    // A row is cut on both sides where the dropped entries can add at most 0.5e-18 max|y| to a value of the spline:
    // |r_j| <= 2 max|y| (1/h_j + 1/h_{j-1}), and M_i enters a value with a weight of at most 0.385 max(h_{i-1}, h_i)^2 / 6.
    if (n >= 3 && n <= BAND_MAX_KNOTS) {
        std::vector<long double> hh(n, 0.0L), a(n, 0.0L), cc(n, 0.0L), dt(n, 0.0L), db(n, 0.0L), g(n, 0.0L), row(n, 0.0L);   // interior rows 1 .. n-2
        for (int i = 0; i + 1 < n; ++i) hh[i] = (long double)(l_list[i + 1] - l_list[i]);
        for (int i = 1; i < n - 1; ++i) { a[i] = (hh[i - 1] + hh[i]) / 3.0L; g[i] = 2.0L * (1.0L / hh[i] + 1.0L / hh[i - 1]); }
        for (int i = 1; i < n - 2; ++i) cc[i] = hh[i] / 6.0L;
        dt[1] = a[1];
        for (int i = 2; i < n - 1; ++i) dt[i] = a[i] - cc[i - 1] * cc[i - 1] / dt[i - 1];
        db[n - 2] = a[n - 2];
        for (int i = n - 3; i >= 1; --i) db[i] = a[i] - cc[i] * cc[i] / db[i + 1];
        std::vector<double> ainv;
        std::vector<int32_t> a_off(n, 0), a_lo(n, 0), a_cnt(n, 0);
        for (int i = 1; i < n - 1; ++i) {
            const long double hm = std::max(hh[i - 1], hh[i]);
            const long double budget = 0.5e-18L / (0.385L * hm * hm / 6.0L);
            // the row outward from the diagonal, as far as its entries stay above 1e-300 (they fall monotonically:
            // what lies beyond is below that and counts as zero)
            row[i] = 1.0L / (dt[i] + db[i] - a[i]);
            int hi = i, lo = i;
            while (hi + 1 <= n - 2 && fabsl(row[hi]) > 1e-300L) { row[hi + 1] = -(cc[hi] / db[hi + 1]) * row[hi]; ++hi; }
            while (lo - 1 >= 1 && fabsl(row[lo]) > 1e-300L) { row[lo - 1] = -(cc[lo - 1] / dt[lo - 1]) * row[lo]; --lo; }
            long double tail = 0.0L;
            while (hi > i && tail + fabsl(row[hi]) * g[hi] <= budget) { tail += fabsl(row[hi]) * g[hi]; --hi; }
            tail = 0.0L;
            while (lo < i && tail + fabsl(row[lo]) * g[lo] <= budget) { tail += fabsl(row[lo]) * g[lo]; ++lo; }
            a_off[i] = (int32_t)ainv.size(); a_lo[i] = lo; a_cnt[i] = hi - lo + 1;
            for (int j = lo; j <= hi; ++j) ainv.push_back((double)row[j]);
        }
        GCAMB_CUDA(cudaMalloc(&p->d_sp_ainv, sizeof(double) * std::max<size_t>(ainv.size(), 1)));
        GCAMB_CUDA(cudaMalloc(&p->d_sp_aoff, sizeof(int32_t) * n));
        GCAMB_CUDA(cudaMalloc(&p->d_sp_alo, sizeof(int32_t) * n));
        GCAMB_CUDA(cudaMalloc(&p->d_sp_acnt, sizeof(int32_t) * n));
        GCAMB_CUDA(cudaMemcpyAsync(p->d_sp_ainv, ainv.data(), sizeof(double) * ainv.size(), cudaMemcpyHostToDevice, stream));
        GCAMB_CUDA(cudaMemcpyAsync(p->d_sp_aoff, a_off.data(), sizeof(int32_t) * n, cudaMemcpyHostToDevice, stream));
        GCAMB_CUDA(cudaMemcpyAsync(p->d_sp_alo, a_lo.data(), sizeof(int32_t) * n, cudaMemcpyHostToDevice, stream));
        GCAMB_CUDA(cudaMemcpyAsync(p->d_sp_acnt, a_cnt.data(), sizeof(int32_t) * n, cudaMemcpyHostToDevice, stream));
        GCAMB_CUDA(cudaStreamSynchronize(stream));
    }
    GCAMB_CUDA(cudaStreamSynchronize(stream));   // the vectors die with this scope
    return GCAMB_OK;
}

gcamb_status launch_cl_interp(const gcamb_los_plan *p, int n_batch, const double *Cl_samp, double *Cl_all,
                              cudaStream_t stream)
{
    if (p->n_l_out < 2) { set_error("interpolation in l needs at least two multipoles in the plan's l list"); return GCAMB_EINVAL; }
    const size_t smem = (sizeof(double) * 2 + sizeof(int)) * (size_t)p->n_l_out;
    if (smem > INTERP_SMEM_MAX) {
        set_error("interpolation in l: n_l = %d exceeds %d knots", p->n_l_out, (int)(INTERP_SMEM_MAX / 20));
        return GCAMB_EINVAL;
    }
    if (smem > 48 * 1024)
        GCAMB_CUDA(cudaFuncSetAttribute(cl_interp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const long long series = (long long)n_batch * p->n_spec;
    const int n_all = p->l_user_last - p->l_user_first + 1;
    if (p->d_sp_ainv) {   // short lists: banded inverse, evaluation spread over thread blocks
        const size_t smem_b = (sizeof(double) * 3 + sizeof(int)) * (size_t)p->n_l_out;   // <= 56 KB at 2048 knots
        static std::atomic<unsigned long long> attr_done{0};
        const unsigned long long dev_bit = 1ull << (p->device & 63);
        if (smem_b > 48 * 1024 && !(attr_done.load(std::memory_order_acquire) & dev_bit)) {
            GCAMB_CUDA(cudaFuncSetAttribute(cl_interp_band_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)((sizeof(double) * 3 + sizeof(int)) * BAND_MAX_KNOTS)));
            attr_done.fetch_or(dev_bit, std::memory_order_release);
        }
        dim3 grid((unsigned)series, (unsigned)((n_all + INTERP_CHUNK - 1) / INTERP_CHUNK));
        cl_interp_band_kernel<<<grid, INTERP_THREADS, smem_b, stream>>>(Cl_samp, Cl_all, p->d_l_user, p->d_sp_seg, p->d_sp_ainv,
                                                                        p->d_sp_aoff, p->d_sp_alo, p->d_sp_acnt, p->n_l_out, n_all);
        GCAMB_CUDA(cudaGetLastError());
        return GCAMB_OK;
    }
    cl_interp_kernel<<<(unsigned)series, INTERP_THREADS, smem, stream>>>(
        Cl_samp, Cl_all, p->d_l_user, p->d_sp_seg, p->d_sp_mult, p->d_sp_inv_diag, p->n_l_out,
        n_all);
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

}  // namespace gcamb
