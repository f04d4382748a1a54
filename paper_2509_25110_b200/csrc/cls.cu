// cls.cu -- step a4: C_l^{XY} = 4 pi sum_j dlnk_j P_R(k_j) Delta^X_l(k_j) Delta^Y_l(k_j)
// (Eq. 1; discrete form BJ, R6, R12).  HBM-bound: Delta is read exactly once.
//
// Two kernels, chosen by the plan's n_k (and the alignment of the caller's buffers):
//   * cls_stream_kernel (n_k even, <= CLS_STREAM_MAX_K): one persistent CTA per SM walks a contiguous
//     range of (cosmology, l) rows; a producer warp streams the rows of Delta into a shared-memory ring
//     with 1-D TMA bulk copies (cp.async.bulk, completion on mbarriers), STAGES x n_src x <= 12 KB in
//     flight per SM whatever the consumers do; the weights w_j = dlnk_j P_R(k_j) of the current cosmology
//     sit in shared memory, computed once per CTA and cosmology.  The loads of the row-per-CTA kernel
//     below are issued by the threads that consume them, so at config 1 (24 KB rows, 2499 short-lived
//     CTAs) it is bound by load latency: 3.6 TB/s.
//   * cls_kernel: one CTA per (l, cosmology), 16-byte loads, four steps of independent loads in flight
//     per thread.  Long rows (config 4: 160 KB per source) already stream at 6.1 TB/s with it.
// Both: thread-private sums over k in a fixed order, shuffle tree, then the warps in index order:
// deterministic, and a row's result depends neither on the batch nor on the CTA that computes it.
#include <algorithm>
#include <atomic>

#include "los_internal.cuh"
#include "mbar.cuh"

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
                                                          double *__restrict__ Cl, int n_l, int n_k, int te_last)
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
            const int q_out = (te_last && q >= 2) ? 5 - q : q;     // tensor plans: (TT, EE, BB, TE)
            Cl[((size_t)b * NSPEC + q_out) * n_l + l0 + r] = 4.0 * 3.14159265358979323846 * v;
        }
    }
}

// ---- streaming kernel (TMA bulk copies into a shared-memory ring)
constexpr int CLS_STREAM_MAX_K = 6144;    // weights of one cosmology in shared memory: 48 KB
constexpr int CLS_STREAM_CHUNK = 1536;    // k per ring stage and source: 12 KB
__host__ __device__ constexpr int cls_stages(int n_src) { return n_src == 2 ? 6 : 4; }   // ring depth: 144 KB of Delta in flight per SM
constexpr int CLS_CONSUMERS = 256;        // + one producer warp

__device__ __forceinline__ void bulk_load(uint32_t dst_smem, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}

// Rows are flat indices r = b * n_l + li; CTA c takes rows [c R / G, (c+1) R / G).  Every row is cut into
// n_chunks pieces of KC k values (the last one shorter); item = (row, chunk), row-major.
template <int NSRC>
__global__ void __launch_bounds__(CLS_CONSUMERS + 32, 1) cls_stream_kernel(const double *__restrict__ Delta,
                                                                           const double *__restrict__ P_R,
                                                                           const double *__restrict__ dlnk,
                                                                           double *__restrict__ Cl, int n_l, int n_k,
                                                                           long long n_rows, int KC, int n_chunks, int te_last)
{
    constexpr int NSPEC = NSRC + 1, NW = CLS_CONSUMERS / 32, CLS_STAGES = cls_stages(NSRC);
    extern __shared__ __align__(16) double sm_cls[];
    double *wgt = sm_cls;                                           // [n_k] dlnk P_R of the current cosmology
    double *ring = wgt + ((n_k + 1) & ~1);                          // [STAGES][NSRC][KC]
    double *psum = ring + (size_t)CLS_STAGES * NSRC * KC;           // [2][NSPEC][NW]
    const uint32_t bar_full = (uint32_t)__cvta_generic_to_shared(psum + 2 * NSPEC * NW);
    const uint32_t bar_empty = bar_full + 8 * CLS_STAGES;
    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int s = 0; s < CLS_STAGES; ++s) { mbar_init(bar_full + 8 * s, 1); mbar_init(bar_empty + 8 * s, NW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const long long r0 = n_rows * blockIdx.x / gridDim.x, r1 = n_rows * (blockIdx.x + 1) / gridDim.x;
    const long long n_items = (r1 - r0) * n_chunks;

    if (tid >= CLS_CONSUMERS) {
        // ---- producer: one thread keeps the ring full
        if (tid == CLS_CONSUMERS) {
            const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(ring);
            long long row = r0;
            int chunk = 0;
            for (long long it = 0; it < n_items; ++it) {
                const int s = (int)(it % CLS_STAGES);
                if (it >= CLS_STAGES) mbar_wait(bar_empty + 8 * s, (int)((it / CLS_STAGES) - 1) & 1);
                const int len = min(KC, n_k - chunk * KC);
                const uint32_t bytes = (uint32_t)len * 8u;
                mbar_expect_tx(bar_full + 8 * s, bytes * NSRC);
                const long long b = row / n_l, li = row - b * n_l;
#pragma unroll
                for (int q = 0; q < NSRC; ++q)
                    bulk_load(ring_s + (uint32_t)(((size_t)s * NSRC + q) * KC * 8),
                              Delta + (((size_t)b * NSRC + q) * n_l + li) * n_k + (size_t)chunk * KC, bytes,
                              bar_full + 8 * s);
                if (++chunk == n_chunks) { chunk = 0; ++row; }
            }
        }
        return;
    }

    // ---- consumers
    const int lane = tid & 31, warp = tid >> 5;
    long long cur_b = -1;
    long long it = 0;
    for (long long row = r0; row < r1; ++row) {
        const long long b = row / n_l;
        if (b != cur_b) {   // weights of this cosmology (the ring is not touched: the producer runs on)
            asm volatile("bar.sync 1, %0;" ::"n"(CLS_CONSUMERS) : "memory");   // everyone is done with the old weights
            for (int j = tid; j < n_k; j += CLS_CONSUMERS) wgt[j] = dlnk[j] * P_R[(size_t)b * n_k + j];
            asm volatile("bar.sync 1, %0;" ::"n"(CLS_CONSUMERS) : "memory");
            cur_b = b;
        }
        double acc[NSPEC];
#pragma unroll
        for (int q = 0; q < NSPEC; ++q) acc[q] = 0.0;
        for (int chunk = 0; chunk < n_chunks; ++chunk, ++it) {
            const int s = (int)(it % CLS_STAGES);
            const int len = min(KC, n_k - chunk * KC);
            mbar_wait(bar_full + 8 * s, (int)(it / CLS_STAGES) & 1, 64);   // short naps: the data is on its way
            const double2 *w2 = reinterpret_cast<const double2 *>(wgt + (size_t)chunk * KC);
            const double2 *d2 = reinterpret_cast<const double2 *>(ring + (size_t)s * NSRC * KC);
            for (int j = tid; j < len / 2; j += CLS_CONSUMERS) {
                const double2 w = w2[j], t = d2[j], e = d2[KC / 2 + j];
                acc[0] = fma(w.x * t.x, t.x, acc[0]);
                acc[1] = fma(w.x * e.x, e.x, acc[1]);
                acc[2] = fma(w.x * t.x, e.x, acc[2]);
                acc[0] = fma(w.y * t.y, t.y, acc[0]);
                acc[1] = fma(w.y * e.y, e.y, acc[1]);
                acc[2] = fma(w.y * t.y, e.y, acc[2]);
                if (NSRC == 3) {
                    const double2 ph = d2[(NSRC - 1) * (KC / 2) + j];
                    acc[NSPEC - 1] = fma(w.x * ph.x, ph.x, acc[NSPEC - 1]);
                    acc[NSPEC - 1] = fma(w.y * ph.y, ph.y, acc[NSPEC - 1]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * s);
        }
        // warps in index order (fixed); the partial sums are double-buffered by row parity, so one
        // barrier per row suffices
        double *ps = psum + (size_t)((row - r0) & 1) * NSPEC * NW;
#pragma unroll
        for (int q = 0; q < NSPEC; ++q) {
            double v = acc[q];
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) ps[q * NW + warp] = v;
        }
        asm volatile("bar.sync 1, %0;" ::"n"(CLS_CONSUMERS) : "memory");
        if (tid < NSPEC) {
            double v = 0.0;
#pragma unroll
            for (int wv = 0; wv < NW; ++wv) v += ps[tid * NW + wv];
            const long long li = row - b * n_l;
            // tensor plans write (TT, EE, BB, TE): the cross spectrum last
            const int q_out = (te_last && tid >= 2) ? 5 - tid : tid;
            Cl[((size_t)b * NSPEC + q_out) * n_l + li] = 4.0 * 3.14159265358979323846 * v;
        }
    }
}

static size_t cls_stream_smem(int n_src, int n_k, int KC)
{
    return sizeof(double) * (((size_t)n_k + 1) & ~(size_t)1) + sizeof(double) * (size_t)cls_stages(n_src) * n_src * KC +
           sizeof(double) * 2 * (n_src + 1) * (CLS_CONSUMERS / 32) + 8 * 2 * cls_stages(n_src);
}

template <int NSRC, int R, int THREADS>
static void launch_rows(bool vec, dim3 grid, cudaStream_t stream, const double *Delta, const double *P_R,
                        const double *dlnk, double *Cl, int n_l, int n_k, int te_last)
{
    if (vec) cls_kernel<NSRC, R, 2, THREADS><<<grid, THREADS, 0, stream>>>(Delta, P_R, dlnk, Cl, n_l, n_k, te_last);
    else cls_kernel<NSRC, R, 1, THREADS><<<grid, THREADS, 0, stream>>>(Delta, P_R, dlnk, Cl, n_l, n_k, te_last);
}

gcamb_status launch_cls(const gcamb_los_plan *p, int n_batch, const double *Delta,
                        const double *P_R, double *Cl, cudaStream_t stream)
{
    // 16-byte loads need even rows and aligned bases (every row then starts on a 16-byte boundary)
    const bool vec = p->n_k % 2 == 0 && ((uintptr_t)Delta | (uintptr_t)P_R) % 16 == 0;
    if (p->n_k % 2 == 0 && (uintptr_t)Delta % 16 == 0 && p->n_k <= CLS_STREAM_MAX_K) {
        const int n_chunks = (p->n_k + CLS_STREAM_CHUNK - 1) / CLS_STREAM_CHUNK;
        const int KC = (((p->n_k + n_chunks - 1) / n_chunks) + 1) & ~1;      // even: every chunk starts 16-byte aligned
        const long long n_rows = (long long)n_batch * p->n_l_out;
        const unsigned grid = (unsigned)std::min<long long>(n_rows, p->n_sm);
        const size_t smem = cls_stream_smem(p->n_src, p->n_k, KC);
        auto kern = p->n_src == 2 ? cls_stream_kernel<2> : cls_stream_kernel<3>;
        static std::atomic<unsigned long long> attr_done[2];
        const unsigned long long dev_bit = 1ull << (p->device & 63);
        if (!(attr_done[p->n_src - 2].load(std::memory_order_acquire) & dev_bit)) {
            GCAMB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)cls_stream_smem(p->n_src, CLS_STREAM_MAX_K, CLS_STREAM_CHUNK)));
            attr_done[p->n_src - 2].fetch_or(dev_bit, std::memory_order_release);
        }
        kern<<<grid, CLS_CONSUMERS + 32, smem, stream>>>(Delta, P_R, p->d_dlnk, Cl, p->n_l_out, p->n_k, n_rows, KC, n_chunks, p->tensor);
        GCAMB_CUDA(cudaGetLastError());
        return GCAMB_OK;
    }
    int R = CLS_ROWS, threads = CLS_THREADS_DEFAULT;
    // few rows: one row per CTA keeps more SMs busy
    while (R > 1 && (long long)((p->n_l_out + R - 1) / R) * n_batch < 2LL * p->n_sm) R >>= 1;
    dim3 grid((unsigned)((p->n_l_out + R - 1) / R), (unsigned)n_batch);
#define GCAMB_CLS(NS, RR, TH) launch_rows<NS, RR, TH>(vec, grid, stream, Delta, P_R, p->d_dlnk, Cl, p->n_l_out, p->n_k, p->tensor)
#define GCAMB_CLS_R(NS, TH) do { if (R == 4) GCAMB_CLS(NS, 4, TH); else if (R == 2) GCAMB_CLS(NS, 2, TH); else GCAMB_CLS(NS, 1, TH); } while (0)
    if (p->n_src == 2) { if (threads == 128) GCAMB_CLS_R(2, 128); else GCAMB_CLS_R(2, 256); }
    else               { if (threads == 128) GCAMB_CLS_R(3, 128); else GCAMB_CLS_R(3, 256); }
#undef GCAMB_CLS_R
#undef GCAMB_CLS
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

}  // namespace gcamb
