// transfer.cu -- steps a1-a3 of the hot path: sources -> Delta^X_l(k)  (Eq. 2-3).
//
// Mapping: one CTA per k (per tau-split), lanes <-> consecutive tau.
// Every thread carries T (k,tau) points ("slots") whose recurrence state lives in registers for
// the whole walk: f_{l+1}, f_l, 1/x and the pre-weighted sources s_X = w S_X (s_E also / x^2).
// The CTA walks l DOWNWARD in tiles of V; per point and l it issues
//     c   = (2l+1) * (1/x)                  1 DMUL
//     acc_X[l] += s_X * f_l                 n_src DFMA
//     f_{l-1} = c * f_l - f_{l+1}           1 DFMA
// i.e. 2 + n_src FP64 issue slots per executed (l,k,tau) term, no j_l table, no sincos: the start
// pair of each point comes from the plan (plan.cu).  After a tile the V x n_src per-thread sums
// are reduced across the warp with a transposing butterfly (1 DADD + 1 double SHFL per l and
// source), across warps through shared memory, scaled (Delta^E prefactor) and stored.
// Points whose cut L(x) lies below the current tile are not walked at all (R16): whole slots
// are skipped with a warp-uniform branch, single lanes are predicated off.
#include "los_internal.cuh"

namespace gcamb {

struct TransferParams {
    const double *S[3];
    double *Delta;
    const double *k, *chi, *w, *pref;
    const double2 *start;
    const int32_t *tile, *korder, *l_index;
    int n_k, n_tau, n_l, l_min, l_max, n_tiles, n_batch, n_split, split_len;
};

constexpr unsigned FULL = 0xffffffffu;

// a[s] (s < V) per lane  ->  sum over the 32 lanes of a[s], returned on every lane for
// s = lane / (32 / V).  V/2 + V/4 + ... + 1 exchanges, then log2(32/V) plain butterfly steps.
template <int V>
__device__ __forceinline__ double warp_transpose_reduce(double (&a)[V], int lane)
{
    int bit = 16;
#pragma unroll
    for (int h = V / 2; h >= 1; h >>= 1, bit >>= 1) {
        const bool up = (lane & bit) != 0;
#pragma unroll
        for (int i = 0; i < h; ++i) {
            const double send = up ? a[i] : a[i + h];
            const double keep = up ? a[i + h] : a[i];
            a[i] = keep + __shfl_xor_sync(FULL, send, bit);
        }
    }
#pragma unroll
    for (; bit >= 1; bit >>= 1) a[0] += __shfl_xor_sync(FULL, a[0], bit);
    return a[0];
}

template <int T, int V, int NSRC, int MAXTHREADS, int MINBLOCKS>
__global__ void __launch_bounds__(MAXTHREADS, MINBLOCKS) transfer_kernel(const TransferParams p)
{
    extern __shared__ double red[];  // [2][W][NSRC][V]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, W = blockDim.x >> 5;
    const int bid = blockIdx.x;
    const int krank = bid / p.n_batch, b = bid - krank * p.n_batch;
    const int kidx = p.korder[krank];
    const int split = blockIdx.y;
    const int i_begin = split * p.split_len;
    const int i_end = min(p.n_tau, i_begin + p.split_len);
    const double kval = p.k[kidx];

    // ---- a1: source staging.  slot j of this thread is tau index i_begin + j*blockDim + tid.
    double fa[T], fb[T], ix[T], src[NSRC][T];
    int tp[T];
    int tall = -1;   // last start tile among this thread's valid points
    int nslot = 0;   // slots of this WARP that hold at least one valid point (warp-uniform)
#pragma unroll
    for (int j = 0; j < T; ++j) {
        const int i = i_begin + j * (int)blockDim.x + tid;
        if (i - lane < i_end) nslot = j + 1;
        if (i < i_end) {
            const size_t pt = (size_t)kidx * p.n_tau + i;
            const size_t sx = ((size_t)b * p.n_k + kidx) * p.n_tau + i;
            const double x = __dmul_rn(kval, p.chi[i]);
            const double inv = 1.0 / x;
            const double w = p.w[i];
            const double2 st = p.start[pt];
            fa[j] = st.x;
            fb[j] = st.y;
            ix[j] = inv;
            tp[j] = p.tile[pt];
            tall = max(tall, tp[j]);
            src[0][j] = w * p.S[0][sx];
            src[1][j] = w * p.S[1][sx] * (inv * inv);
            if (NSRC == 3) src[NSRC - 1][j] = w * p.S[2][sx];
        } else {
            fa[j] = fb[j] = ix[j] = 0.0;
            tp[j] = 0x7fffffff;
#pragma unroll
            for (int q = 0; q < NSRC; ++q) src[q][j] = 0.0;
        }
    }
    tall = __reduce_max_sync(FULL, tall);
    const bool warp_full = nslot == T;

    // first tile of this CTA = start tile of its largest x (tau is increasing, x decreasing)
    const int t_begin = p.tile[(size_t)kidx * p.n_tau + i_begin];
    const size_t delta_b = (size_t)b * NSRC * p.n_l;

    // l above the first tile: Delta is exactly zero there (R16).  With RED output the buffer was
    // zeroed by the launcher instead.
    if (p.n_split == 1) {
        const int l_top = p.l_max - t_begin * V;  // highest l walked
        for (int l = p.l_max - tid; l > l_top; l -= blockDim.x) {
            const int li = p.l_index[l];
            if (li >= 0) {
#pragma unroll
                for (int q = 0; q < NSRC; ++q) p.Delta[(delta_b + (size_t)q * p.n_l + li) * p.n_k + kidx] = 0.0;
            }
        }
    }

    int buf = 0;
    for (int t = t_begin; t < p.n_tiles; ++t) {
        const int lhi = p.l_max - t * V;
        const double tl0 = (double)(2 * lhi + 1);
        double acc[NSRC][V];
#pragma unroll
        for (int q = 0; q < NSRC; ++q)
#pragma unroll
            for (int s = 0; s < V; ++s) acc[q][s] = 0.0;

        if (warp_full && t >= tall) {
            // ---- a2 + a3, steady state: every point of the warp is active; T independent chains
#pragma unroll
            for (int s = 0; s < V; ++s) {
                const double tl = tl0 - 2.0 * s;
#pragma unroll
                for (int j = 0; j < T; ++j) {
                    const double c = tl * ix[j];
#pragma unroll
                    for (int q = 0; q < NSRC; ++q) acc[q][s] = fma(src[q][j], fb[j], acc[q][s]);
                    const double fn = fma(c, fb[j], -fa[j]);
                    fa[j] = fb[j];
                    fb[j] = fn;
                }
            }
        } else {
            // ---- ragged top: skip slots that have not started, predicate single lanes
#pragma unroll
            for (int j = 0; j < T; ++j) {
                if (j < nslot && __any_sync(FULL, t >= tp[j])) {
                    if (t >= tp[j]) {
#pragma unroll
                        for (int s = 0; s < V; ++s) {
                            const double c = (tl0 - 2.0 * s) * ix[j];
#pragma unroll
                            for (int q = 0; q < NSRC; ++q) acc[q][s] = fma(src[q][j], fb[j], acc[q][s]);
                            const double fn = fma(c, fb[j], -fa[j]);
                            fa[j] = fb[j];
                            fb[j] = fn;
                        }
                    }
                }
            }
        }

        // ---- cross-thread reduction: warp butterfly, then warps through shared memory
        double *rb = red + (size_t)buf * W * NSRC * V;
#pragma unroll
        for (int q = 0; q < NSRC; ++q) {
            const double tot = warp_transpose_reduce<V>(acc[q], lane);
            if ((lane & (32 / V - 1)) == 0) rb[(warp * NSRC + q) * V + lane / (32 / V)] = tot;
        }
        __syncthreads();
        for (int idx = tid; idx < NSRC * V; idx += blockDim.x) {
            const int q = idx / V, s = idx - q * V;
            const int l = lhi - s;
            if (l >= p.l_min) {
                const int li = p.l_index[l];
                if (li >= 0) {
                    double sum = 0.0;
                    for (int wv = 0; wv < W; ++wv) sum += rb[(wv * NSRC + q) * V + s];
                    if (q == 1) sum *= p.pref[li];
                    double *dst = p.Delta + (delta_b + (size_t)q * p.n_l + li) * p.n_k + kidx;
                    if (p.n_split == 1) *dst = sum;
                    else atomicAdd(dst, sum);
                }
            }
        }
        buf ^= 1;
    }
}

// ------------------------------------------------------------------------------------------
TransferShape choose_shape(int n_tau, int n_src)
{
    TransferShape s;
    s.T = 8;
    s.V = n_src == 2 ? 16 : 8;
    const int max_threads = n_src == 2 ? 384 : 320;   // register file: threads * regs <= 64K
    s.n_split = 1;
    for (;;) {
        const int len = (n_tau + s.n_split - 1) / s.n_split;
        const int threads = ((len + s.T - 1) / s.T + 31) / 32 * 32;
        if (threads <= max_threads) { s.threads = threads; break; }
        ++s.n_split;
    }
    return s;
}

template <int T, int V, int NSRC, int MAXT, int MINB>
static gcamb_status launch_impl(const TransferParams &prm, const TransferShape &sh, cudaStream_t stream)
{
    dim3 grid((unsigned)(prm.n_k * prm.n_batch), (unsigned)sh.n_split);
    const size_t smem = sizeof(double) * 2 * (sh.threads / 32) * NSRC * V;
    transfer_kernel<T, V, NSRC, MAXT, MINB><<<grid, sh.threads, smem, stream>>>(prm);
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

gcamb_status launch_transfer(const gcamb_los_plan *p, int n_batch, const double *S_T,
                             const double *S_E, const double *S_phi, double *Delta,
                             cudaStream_t stream)
{
    const TransferShape &sh = p->shape;
    TransferParams prm;
    prm.S[0] = S_T; prm.S[1] = S_E; prm.S[2] = S_phi;
    prm.Delta = Delta;
    prm.k = p->d_k; prm.chi = p->d_chi; prm.w = p->d_w; prm.pref = p->d_pref;
    prm.start = p->d_start; prm.tile = p->d_tile; prm.korder = p->d_korder; prm.l_index = p->d_l_index;
    prm.n_k = p->n_k; prm.n_tau = p->n_tau; prm.n_l = p->n_l;
    prm.l_min = p->l_min; prm.l_max = p->l_max; prm.n_tiles = p->n_tiles;
    prm.n_batch = n_batch; prm.n_split = sh.n_split;
    prm.split_len = (p->n_tau + sh.n_split - 1) / sh.n_split;
    if (sh.n_split > 1) {
        const size_t bytes = sizeof(double) * (size_t)n_batch * p->n_src * p->n_l * p->n_k;
        GCAMB_CUDA(cudaMemsetAsync(Delta, 0, bytes, stream));
    }
    if (p->n_src == 2 && sh.T == 8 && sh.V == 16) return launch_impl<8, 16, 2, 384, 1>(prm, sh, stream);
    if (p->n_src == 3 && sh.T == 8 && sh.V == 8) return launch_impl<8, 8, 3, 320, 1>(prm, sh, stream);
    set_error("no transfer kernel for T=%d V=%d n_src=%d", sh.T, sh.V, p->n_src);
    return GCAMB_EINVAL;
}

}  // namespace gcamb
