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
//   solve:  one thread per (series, tau) walks the coarse grid down and up (two dependent FMA chains of
//           n_kc steps; the loads do not depend on the chain), second derivatives M to scratch;
//   eval:   one thread per (series, k, tau): four coarse values (L2-resident) -> one fine value, the
//           HBM-bound part (8 n_k n_tau bytes written per series).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <new>
#include <vector>

#include "los_internal.cuh"

struct gcamb_los_srcinterp {
    int32_t n_kc, n_k, n_tau, device;
    double *d_h;          // [n_kc]   h_i = kc_{i+1} - kc_i (last entry unused)
    double *d_ih;         // [n_kc]   1 / h_i (an fp64 division is ~40 dependent instructions: none in the sweeps)
    double *d_mult;       // [n_kc]   forward-elimination multipliers
    double *d_inv_diag;   // [n_kc]   reciprocals of the eliminated diagonal
    int32_t *d_seg;       // [n_k]    coarse interval of every fine k
    double4 *d_wgt;       // [n_k]    (A, B, (A^3-A) h^2/6, (B^3-B) h^2/6)
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

constexpr int EVAL_ROWS = 8;   // fine k rows per CTA (one row per CTA: 30000 one-shot CTAs, 33 us for 58 MB)

__global__ void __launch_bounds__(256) srcinterp_eval_kernel(const double *__restrict__ S_c, const double *__restrict__ M,
                                                             const int32_t *__restrict__ seg, const double4 *__restrict__ wgt,
                                                             double *__restrict__ S_f, int n_kc, int n_k, int n_tau)
{
    const size_t cbase = (size_t)blockIdx.z * n_kc * n_tau;
    const int j_end = min(n_k, (int)(blockIdx.y + 1) * EVAL_ROWS);
    for (int j = blockIdx.y * EVAL_ROWS; j < j_end; ++j) {
        const size_t fbase = ((size_t)blockIdx.z * n_k + j) * n_tau;
        const int s = seg[j];
        const double4 w = wgt[j];
        const double *y0 = S_c + cbase + (size_t)s * n_tau, *m0 = M + cbase + (size_t)s * n_tau;
        for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < n_tau; t += gridDim.x * blockDim.x)
            S_f[fbase + t] = w.x * y0[t] + w.y * y0[n_tau + t] + (w.z * m0[t] + w.w * m0[n_tau + t]);
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
    if (cur >= 0 && cur != si->device) cudaSetDevice(cur);
    delete si;
    if (e != cudaSuccess) return cuda_fail(e, "gcamb_los_srcinterp_destroy");
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
    dim3 g2((unsigned)std::min((si->n_tau + 255) / 256, 16), (unsigned)((si->n_k + EVAL_ROWS - 1) / EVAL_ROWS), (unsigned)n_series);
    srcinterp_eval_kernel<<<g2, 256, 0, s>>>(d_S_coarse, d_work, si->d_seg, si->d_wgt, d_S_fine, si->n_kc, si->n_k, si->n_tau);
    GCAMB_CUDA(cudaGetLastError());
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
