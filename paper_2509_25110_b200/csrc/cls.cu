// cls.cu -- step a4: C_l^{XY} = 4 pi sum_j dlnk_j P_R(k_j) Delta^X_l(k_j) Delta^Y_l(k_j)
// (Eq. 1; discrete form BJ, R6, R12).  HBM-bound: Delta is read exactly once,
// coalesced along k with 16-byte loads, four steps of 2 + R n_src independent loads in flight per
// thread.  One CTA takes R consecutive l of one cosmology (R = 1: see CLS_ROWS below).  Fixed-order
// (deterministic) reduction: thread-private sums over k, shuffle tree, then the warps in index order.
#include "los_internal.cuh"

namespace gcamb {

// Measured on B200 (profiles/README.md, cls section): one row per 256-thread CTA is the fastest shape at
// every config (rows per CTA 1 / 2 / 4 at config 1: 35 / 39 / 45 us; at config 4: 0.70 / 0.84 / 0.99 ms):
// more rows per CTA mean fewer, longer-lived CTAs and a coarser tail.
constexpr int CLS_ROWS = 1;               // l rows per CTA (rows of a CTA share the weights)
constexpr int CLS_THREADS_DEFAULT = 256;

template <int VEC> struct Pack;
template <> struct Pack<1> { double v[1]; };
template <> struct alignas(16) Pack<2> { double v[2]; };

template <int NSRC, int R, int VEC, int CLS_THREADS>
__global__ void __launch_bounds__(CLS_THREADS) cls_kernel(const double *__restrict__ Delta,
                                                          const double *__restrict__ P_R,
                                                          const double *__restrict__ dlnk,
                                                          double *__restrict__ Cl, int n_l, int n_k)
{
    constexpr int NSPEC = NSRC + 1;
    using pack = Pack<VEC>;
    const int l0 = blockIdx.x * R, b = blockIdx.y;
    const pack *row[R][NSRC];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int li = min(l0 + r, n_l - 1);   // rows past the end re-read the last one and are dropped below
#pragma unroll
        for (int q = 0; q < NSRC; ++q)
            row[r][q] = reinterpret_cast<const pack *>(Delta + (((size_t)b * NSRC + q) * n_l + li) * n_k);
    }
    const pack *pr = reinterpret_cast<const pack *>(P_R + (size_t)b * n_k);
    const pack *dl = reinterpret_cast<const pack *>(dlnk);
    double s[R][NSPEC];
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int q = 0; q < NSPEC; ++q) s[r][q] = 0.0;
    const int n_pack = n_k / VEC;
#pragma unroll 4
    for (int j = threadIdx.x; j < n_pack; j += CLS_THREADS) {
        const pack a = dl[j], c = pr[j];
        pack d[R][NSRC];
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int q = 0; q < NSRC; ++q) d[r][q] = row[r][q][j];
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            const double wp = a.v[v] * c.v[v];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double t = d[r][0].v[v], e = d[r][1].v[v];
                s[r][0] = fma(wp * t, t, s[r][0]);
                s[r][1] = fma(wp * e, e, s[r][1]);
                s[r][2] = fma(wp * t, e, s[r][2]);
                if (NSRC == 3) {
                    const double ph = d[r][NSRC - 1].v[v];
                    s[r][NSPEC - 1] = fma(wp * ph, ph, s[r][NSPEC - 1]);
                }
            }
        }
    }
    __shared__ double sm[R * NSPEC][CLS_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int q = 0; q < NSPEC; ++q) {
            double v = s[r][q];
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) sm[r * NSPEC + q][warp] = v;
        }
    __syncthreads();
    if (threadIdx.x < R * NSPEC) {
        const int r = threadIdx.x / NSPEC, q = threadIdx.x - r * NSPEC;
        if (l0 + r < n_l) {
            double v = 0.0;
#pragma unroll
            for (int wv = 0; wv < CLS_THREADS / 32; ++wv) v += sm[threadIdx.x][wv];
            Cl[((size_t)b * NSPEC + q) * n_l + l0 + r] = 4.0 * 3.14159265358979323846 * v;
        }
    }
}

template <int NSRC, int R, int THREADS>
static void launch_rows(bool vec, dim3 grid, cudaStream_t stream, const double *Delta, const double *P_R,
                        const double *dlnk, double *Cl, int n_l, int n_k)
{
    if (vec) cls_kernel<NSRC, R, 2, THREADS><<<grid, THREADS, 0, stream>>>(Delta, P_R, dlnk, Cl, n_l, n_k);
    else cls_kernel<NSRC, R, 1, THREADS><<<grid, THREADS, 0, stream>>>(Delta, P_R, dlnk, Cl, n_l, n_k);
}

gcamb_status launch_cls(const gcamb_los_plan *p, int n_batch, const double *Delta,
                        const double *P_R, double *Cl, cudaStream_t stream)
{
    // 16-byte loads need even rows and aligned bases (every row then starts on a 16-byte boundary)
    const bool vec = p->n_k % 2 == 0 && ((uintptr_t)Delta | (uintptr_t)P_R) % 16 == 0;
    int R = CLS_ROWS, threads = CLS_THREADS_DEFAULT;
    // few rows: one row per CTA keeps more SMs busy
    while (R > 1 && (long long)((p->n_l + R - 1) / R) * n_batch < 2LL * p->n_sm) R >>= 1;
    dim3 grid((unsigned)((p->n_l + R - 1) / R), (unsigned)n_batch);
#define GCAMB_CLS(NS, RR, TH) launch_rows<NS, RR, TH>(vec, grid, stream, Delta, P_R, p->d_dlnk, Cl, p->n_l, p->n_k)
#define GCAMB_CLS_R(NS, TH) do { if (R == 4) GCAMB_CLS(NS, 4, TH); else if (R == 2) GCAMB_CLS(NS, 2, TH); else GCAMB_CLS(NS, 1, TH); } while (0)
    if (p->n_src == 2) { if (threads == 128) GCAMB_CLS_R(2, 128); else GCAMB_CLS_R(2, 256); }
    else               { if (threads == 128) GCAMB_CLS_R(3, 128); else GCAMB_CLS_R(3, 256); }
#undef GCAMB_CLS_R
#undef GCAMB_CLS
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

}  // namespace gcamb
