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
// once.  A call does, per (cosmology, spectrum), one thread block:
//     y_i, right-hand sides                      all threads
//     forward sweep, back substitution           one thread: two dependent FMA chains of n_l steps
//                                                (n_l ~ 100 for a CAMB-like list: ~1 us)
//     s(l) = A y_i + B y_{i+1} + ((A^3-A) M_i + (B^3-B) M_{i+1}) h_i^2/6 on every integer l,
//     A = (l_{i+1}-l)/h_i, B = (l-l_i)/h_i       all threads, coalesced stores
// Deterministic: no atomics, the order of every operation is fixed.
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
    cl_interp_kernel<<<(unsigned)series, INTERP_THREADS, smem, stream>>>(
        Cl_samp, Cl_all, p->d_l_user, p->d_sp_seg, p->d_sp_mult, p->d_sp_inv_diag, p->n_l_out,
        p->l_max - p->tensor - p->l_min + 1);
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

}  // namespace gcamb
