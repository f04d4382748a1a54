// cls.cu -- step a4: C_l^{XY} = 4 pi sum_j dlnk_j P_R(k_j) Delta^X_l(k_j) Delta^Y_l(k_j)
// (Eq. 1; discrete form BJ, R6, R12).  HBM-bound: Delta is read exactly once,
// coalesced along k; one CTA per (l, cosmology); fixed-order (deterministic) block reduction.
#include "los_internal.cuh"

namespace gcamb {

constexpr int CLS_THREADS = 256;

template <int NSRC>
__global__ void __launch_bounds__(CLS_THREADS) cls_kernel(const double *__restrict__ Delta,
                                                          const double *__restrict__ P_R,
                                                          const double *__restrict__ dlnk,
                                                          double *__restrict__ Cl, int n_l, int n_k)
{
    constexpr int NSPEC = NSRC + 1;
    const int li = blockIdx.x, b = blockIdx.y;
    const double *dT = Delta + (((size_t)b * NSRC + 0) * n_l + li) * n_k;
    const double *dE = Delta + (((size_t)b * NSRC + 1) * n_l + li) * n_k;
    const double *dP = NSRC == 3 ? Delta + (((size_t)b * NSRC + 2) * n_l + li) * n_k : nullptr;
    const double *pr = P_R + (size_t)b * n_k;
    double s[NSPEC];
#pragma unroll
    for (int q = 0; q < NSPEC; ++q) s[q] = 0.0;
    for (int j = threadIdx.x; j < n_k; j += CLS_THREADS) {
        const double wp = dlnk[j] * pr[j];
        const double t = dT[j], e = dE[j];
        s[0] = fma(wp * t, t, s[0]);
        s[1] = fma(wp * e, e, s[1]);
        s[2] = fma(wp * t, e, s[2]);
        if (NSRC == 3) {
            const double ph = dP[j];
            s[NSPEC - 1] = fma(wp * ph, ph, s[NSPEC - 1]);
        }
    }
    __shared__ double sm[NSPEC][CLS_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < NSPEC; ++q) {
        double v = s[q];
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) sm[q][warp] = v;
    }
    __syncthreads();
    if (threadIdx.x < NSPEC) {
        double v = 0.0;
#pragma unroll
        for (int wv = 0; wv < CLS_THREADS / 32; ++wv) v += sm[threadIdx.x][wv];
        Cl[((size_t)b * NSPEC + threadIdx.x) * n_l + li] = 4.0 * 3.14159265358979323846 * v;
    }
}

gcamb_status launch_cls(const gcamb_los_plan *p, int n_batch, const double *Delta,
                        const double *P_R, double *Cl, cudaStream_t stream)
{
    dim3 grid((unsigned)p->n_l, (unsigned)n_batch);
    if (p->n_src == 2)
        cls_kernel<2><<<grid, CLS_THREADS, 0, stream>>>(Delta, P_R, p->d_dlnk, Cl, p->n_l, p->n_k);
    else
        cls_kernel<3><<<grid, CLS_THREADS, 0, stream>>>(Delta, P_R, p->d_dlnk, Cl, p->n_l, p->n_k);
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

}  // namespace gcamb
