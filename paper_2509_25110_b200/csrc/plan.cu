// plan.cu -- device-side precompute of a plan: per-(k,tau) recurrence start values.
//
// For every point x = k (tau0 - tau) the transfer kernel walks l DOWNWARD from the top of the
// first l-tile that is not negligible.  This file computes, once per grid set, that tile index
// and the normalised pair (j_{lhi+1}(x), j_{lhi}(x)) at its top:
//   * cut (R16):   L(x) = ceil(x + 18.2 x^(1/3) + 8);  |j_l(x)| < 1e-36 for l >= L(x)
//   * tiles are anchored at l_max: tile t covers l = l_max - V t ... l_max - V t - V + 1
//   * Miller's backward recurrence (BJ (b)) from M = max(L, lhi) + 50 down to l = 0,
//     f_{l-1} = (2l+1)/x f_l - f_{l+1}, with power-of-two rescaling against overflow,
//   * normalised against the closed forms j_0 = sin x / x and j_1 = (sin x / x - cos x)/x with the
//     two-term least-squares scale of R15 (safe at the zeros of j_0); j_1 by its power series
//     for x < 1 where the closed form cancels.
// For x >= l_max the start is in the oscillatory region, where the downward recurrence is
// neutrally stable (error ~ eps x relative to the envelope, like the forward one).
#include <algorithm>
#include <cmath>
#include <numeric>
#include <queue>
#include <vector>

#include "los_internal.cuh"

namespace gcamb {

__device__ __forceinline__ int l_cut(double x) { return (int)ceil(x + 18.2 * cbrt(x) + 8.0); }

__device__ __forceinline__ double j1_series(double x)
{
    // j_1(x) = x/3 (1 - x^2/10 (1 - x^2/28 (1 - x^2/54 ( ... ))));  ratio -x^2 / (2m(2m+3))
    const double x2 = x * x;
    double term = x / 3.0, sum = term;
    for (int m = 1; m < 30; ++m) {
        term *= -x2 / (double)(2 * m * (2 * m + 3));
        sum += term;
        if (fabs(term) < 1e-18 * fabs(sum)) break;
    }
    return sum;
}

// Open universe (nonflat, reading R28): the radial functions are the hyperspherical Bessel functions
// Phi_l^beta(chi), beta = k r_c, chi = (tau0 - tau)/r_c, with
//   b_{l+1} Phi_{l+1} = (2l+1) coth(chi) Phi_l - b_l Phi_{l-1},   b_l = sqrt(beta^2 + l^2).
// Above the turning point l + 1/2 = beta sinh(chi) the regular solution falls by the smaller root r_l of
// b_{l+1} r^2 - (2l+1) coth(chi) r + b_l = 0 per step (-> tanh(chi/2) for l >> beta, slower than the flat
// j_l when chi is not small): the cut is the first l at which the product of the r_l is below 1e-36, + 8.
// sgn = +1: open (b_l^2 = beta^2 + l^2); sgn = -1: closed (b_l^2 = beta^2 - l^2, integer beta, Phi_l = 0 for
// l >= beta: the cut never exceeds beta - 1, the end of the ladder).
__device__ __forceinline__ double b_curved(double b2, int l, int sgn)
{
    const double v = fma((double)(sgn * l), (double)l, b2);
    return v > 0.0 ? sqrt(v) : 0.0;
}

__device__ __forceinline__ int l_cut_curved(double beta, double cth, double x_turn, int sgn)
{
    int l = max(1, (int)ceil(x_turn));
    const int top = sgn > 0 ? 4000000 : (int)beta - 1;
    double lg = 0.0;
    const double b2 = beta * beta;
    while (lg > -82.9 && l < top) {
        const double bl = b_curved(b2, l, sgn), bl1 = b_curved(b2, l + 1, sgn);
        const double t = (double)(2 * l + 1) * cth;
        const double disc = fma(t, t, -4.0 * bl * bl1);
        if (disc > 0.0) lg += log(2.0 * bl / (t + sqrt(disc)));
        ++l;
    }
    return min(l + 8, top);
}

// CURVED: `chi` holds chi_i = (tau0 - tau_i)/r_c and `k` is multiplied by r_c to give beta; inv_x is not written.
template <bool CURVED>
__global__ void __launch_bounds__(128) start_values_kernel(const double *__restrict__ k,
                                                           const double *__restrict__ chi, int n_tau,
                                                           int l_max, int V, double r_c, int sgn,
                                                           double2 *__restrict__ start,
                                                           int32_t *__restrict__ tile,
                                                           double *__restrict__ inv_x,
                                                           int32_t *__restrict__ cut)
{
    const int i = blockIdx.y * blockDim.x + threadIdx.x;   // k along grid.x: n_k is bounded by 2^31 - 1 only
    const int j = blockIdx.x;
    if (i >= n_tau) return;
    double beta = CURVED ? __dmul_rn(k[j], r_c) : 0.0;
    if (CURVED && sgn < 0) beta = rint(beta);          // closed: integer beta (validated at plan creation)
    const double ch = chi[i];
    const double x = CURVED ? __dmul_rn(beta, ch) : __dmul_rn(k[j], ch);
    const double snh = CURVED ? (sgn > 0 ? sinh(ch) : sin(ch)) : 0.0;
    const double cth = CURVED ? (sgn > 0 ? cosh(ch) : cos(ch)) / snh : 0.0;
    const int L = CURVED ? l_cut_curved(beta, cth, beta * snh, sgn) : l_cut(x);
    const int Ls = min(L, l_max);
    const int t = (l_max - Ls) / V;
    const int lhi = l_max - t * V;  // Ls <= lhi < Ls + V
    // closed: the ladder ends at top = beta - 1 (b_beta = 0).  When the start tile reaches above it, the levels
    // l >= beta are walked with the coefficients (0, -1) of curved_coef_kernel, which keep a constant sequence:
    // the pair handed to the transfer kernel is then (Phi_top, Phi_top), and the flush zeroes Delta_l for l > top.
    const int top = (CURVED && sgn < 0) ? (int)beta - 1 : 0x7fffffff;
    const int M = min(max(L, lhi) + 50, top);
    const int l_cap = min(lhi, top);       // level at which the pair is taken
    if (CURVED) cut[(size_t)j * n_tau + i] = Ls;

    double fa = 0.0, fb = 1.0;  // f_{l+1}, f_l
    double rhi = 0.0, rlo = 0.0;
    int e = 0, re = 0;
    const double b2 = beta * beta;
    double b_up = CURVED ? b_curved(b2, M + 1, sgn) : 0.0;   // b_{l+1}
    for (int l = M; l >= 1; --l) {
        if (l == l_cap) { rlo = fb; rhi = (lhi > top) ? fb : fa; re = e; }
        double fn;
        if (CURVED) {
            const double bl = b_curved(b2, l, sgn);
            fn = ((double)(2 * l + 1) * cth * fb - b_up * fa) / bl;
            b_up = bl;
        } else {
            const double c = (double)(2 * l + 1) / x;
            fn = fma(c, fb, -fa);
        }
        fa = fb;
        fb = fn;
        if (fabs(fb) > 0x1p500) { fa *= 0x1p-500; fb *= 0x1p-500; ++e; }
    }
    // fb = f_0, fa = f_1 (epoch e)
    double s, c;
    sincos(x, &s, &c);
    const double inv = 1.0 / x;
    double j0, j1;
    if (CURVED) {
        // Phi_0 = sin(beta chi)/(beta sinh chi), Phi_1 = (coth sin - beta cos)/(beta sinh chi b_1); for x < 1 the
        // closed form of Phi_1 cancels and Phi_0 ~ 1 alone fixes the scale
        const double d = 1.0 / (beta * snh);
        j0 = s * d;
        j1 = x < 1.0 ? fa * (j0 / fb) : (cth * s - beta * c) * d / b_curved(b2, 1, sgn);
    } else {
        j0 = s * inv;
        j1 = x < 1.0 ? j1_series(x) : (s * inv - c) * inv;
    }
    const double m = fmax(fabs(fb), fabs(fa));
    const double a = fb / m, b = fa / m;
    const double sc = (j0 * a + j1 * b) / ((a * a + b * b) * m);
    int e_sc, e_lo, e_hi;
    const double m_sc = frexp(sc, &e_sc);
    const double m_lo = frexp(rlo, &e_lo);
    const double m_hi = frexp(rhi, &e_hi);
    const int shift = e_sc - 500 * (e - re);
    double2 out;
    out.x = ldexp(m_hi * m_sc, e_hi + shift);
    out.y = ldexp(m_lo * m_sc, e_lo + shift);
    const size_t idx = (size_t)j * n_tau + i;
    start[idx] = out;
    tile[idx] = t;
    if (!CURVED) inv_x[idx] = inv;   // 1/x, correctly rounded: the transfer kernel's coefficient base
}

// Open universe: per (k, l) the two coefficients of a downward step  Phi_{l-1} = A_l coth(chi) Phi_l - R_l Phi_{l+1},
// A_l = (2l+1)/b_l, R_l = b_{l+1}/b_l, laid out as the transfer kernel walks: [k][tile][step], l = l_max - tile V - step
// Closed universes: (0, -1) for l >= beta (see start_values_kernel), R_{beta-1} = b_beta / b_{beta-1} = 0 by itself;
// l_end[k] = beta - 1, the last multipole with a non-zero function (open: none).
__global__ void __launch_bounds__(256) curved_coef_kernel(const double *__restrict__ k, double r_c, int sgn, int l_max, int n_walk,
                                                          double2 *__restrict__ coef, int32_t *__restrict__ l_end)
{
    const int j = blockIdx.y;
    double beta = __dmul_rn(k[j], r_c);
    if (sgn < 0) beta = rint(beta);
    const double b2 = beta * beta;
    if (blockIdx.x == 0 && threadIdx.x == 0) l_end[j] = sgn < 0 ? (int)beta - 1 : 0x7fffffff;
    for (int a = blockIdx.x * blockDim.x + threadIdx.x; a < n_walk; a += gridDim.x * blockDim.x) {
        const int l = l_max - a;
        double2 c = make_double2(0.0, 0.0);
        if (sgn < 0 && (double)l >= beta) {
            c = make_double2(0.0, -1.0);
        } else if (l >= 1) {
            const double bl = b_curved(b2, l, sgn), bl1 = b_curved(b2, l + 1, sgn);
            c = make_double2((double)(2 * l + 1) / bl, bl1 / bl);
        }
        coef[(size_t)j * n_walk + a] = c;
    }
}

// per-k work: walked = sum_i (lhi_i - l_min + 1)+, executed = sum_i (min(L(x_i), l_max) - l_min + 1)+
__global__ void __launch_bounds__(256) k_cost_kernel(const double *__restrict__ k,
                                                     const double *__restrict__ chi, int n_tau,
                                                     int l_min, int l_max, int V,
                                                     const int32_t *__restrict__ tile,
                                                     const int32_t *__restrict__ cut,
                                                     long long *__restrict__ walked,
                                                     long long *__restrict__ executed,
                                                     long long *__restrict__ first_tile)
{
    __shared__ long long sw[256], se[256];
    const int j = blockIdx.x;
    long long w = 0, ex = 0;
    for (int i = threadIdx.x; i < n_tau; i += blockDim.x) {
        const int Ls = cut ? cut[(size_t)j * n_tau + i] : min(l_cut(__dmul_rn(k[j], chi[i])), l_max);
        const int lhi = l_max - tile[(size_t)j * n_tau + i] * V;
        w += max(0, lhi - l_min + 1);
        ex += max(0, Ls - l_min + 1);
    }
    sw[threadIdx.x] = w;
    se[threadIdx.x] = ex;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) {
            sw[threadIdx.x] += sw[threadIdx.x + s];
            se[threadIdx.x] += se[threadIdx.x + s];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { walked[j] = sw[0]; executed[j] = se[0]; first_tile[j] = tile[(size_t)j * n_tau]; }
}

gcamb_status plan_precompute(gcamb_los_plan *p, cudaStream_t stream)
{
    const int V = p->shape.V;
    dim3 grid(p->n_k, (p->n_tau + 127) / 128);
    int32_t *d_cut = nullptr;
    if (p->curved) {
        GCAMB_CUDA(cudaMalloc(&d_cut, sizeof(int32_t) * (size_t)p->n_k * p->n_tau));
        start_values_kernel<true><<<grid, 128, 0, stream>>>(p->d_k, p->d_chi, p->n_tau, p->l_max, V, p->r_c, p->curved,
                                                            p->d_start, p->d_tile, nullptr, d_cut);
        cudaError_t ec = cudaGetLastError();
        if (ec == cudaSuccess) {
            const int n_walk = p->n_tiles * V;
            curved_coef_kernel<<<dim3((unsigned)((n_walk + 255) / 256), (unsigned)p->n_k), 256, 0, stream>>>(
                p->d_k, p->r_c, p->curved, p->l_max, n_walk, p->d_coef, p->d_l_end);
            ec = cudaGetLastError();
        }
        if (ec != cudaSuccess) { cudaFree(d_cut); return cuda_fail(ec, "plan precompute (open universe)"); }
    } else {
        start_values_kernel<false><<<grid, 128, 0, stream>>>(p->d_k, p->d_chi, p->n_tau, p->l_max, V, 0.0, 0,
                                                             p->d_start, p->d_tile, p->d_inv, nullptr);
        GCAMB_CUDA(cudaGetLastError());
    }

    long long *d_cost = nullptr;
    cudaError_t e = cudaMalloc(&d_cost, sizeof(long long) * 3 * (size_t)p->n_k);
    if (e != cudaSuccess) { cudaFree(d_cut); return cuda_fail(e, "plan precompute"); }
    k_cost_kernel<<<p->n_k, 256, 0, stream>>>(p->d_k, p->d_chi, p->n_tau, p->l_min, p->l_max, V,
                                              p->d_tile, d_cut, d_cost, d_cost + p->n_k, d_cost + 2 * p->n_k);
    e = cudaGetLastError();
    std::vector<long long> cost(3 * (size_t)p->n_k);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(cost.data(), d_cost, sizeof(long long) * cost.size(),
                            cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    cudaFree(d_cost);
    cudaFree(d_cut);
    if (e != cudaSuccess) return cuda_fail(e, "plan precompute");

    p->walked_terms = std::accumulate(cost.begin(), cost.begin() + p->n_k, 0LL);
    p->executed_terms = std::accumulate(cost.begin() + p->n_k, cost.begin() + 2 * p->n_k, 0LL);
    // heaviest k first: the CTA scheduler hands out blockIdx in order (longest-processing-time rule)
    std::vector<int32_t> order(p->n_k);
    std::iota(order.begin(), order.end(), 0);
    // ties (saturated rows) by k, so that the order is the k grid reversed whenever cost grows with k
    std::stable_sort(order.begin(), order.end(),
                     [&](int32_t a, int32_t b) { return cost[a] != cost[b] ? cost[a] > cost[b] : a > b; });
    p->order_reversed = 1;
    for (int r = 0; r < p->n_k; ++r) p->order_reversed = p->order_reversed && order[r] == p->n_k - 1 - r;
    GCAMB_CUDA(cudaMemcpyAsync(p->d_korder, order.data(), sizeof(int32_t) * p->n_k,
                               cudaMemcpyHostToDevice, stream));
    // Fused batched path (fused.cu): one static list of k rows per thread-block slot (n_sm of them),
    // balanced by the longest-processing-time rule on the walked terms plus a per-tile and a per-row
    // overhead.  Static lists make the order of the k sum of Eq. 1 independent of the scheduling.
    {
        p->n_bins = p->n_sm;
        const long long per_tile = 700, per_row = 20000;   // in walked-term units (ring + flush per tile; prologue)
        typedef std::pair<long long, int> Load;             // (load, bin): smallest load first
        std::priority_queue<Load, std::vector<Load>, std::greater<Load>> bins;
        for (int b = 0; b < p->n_bins; ++b) bins.push(Load(0, b));
        std::vector<std::vector<int32_t>> items(p->n_bins);
        for (int r = 0; r < p->n_k; ++r) {
            const int j = order[r];
            const long long tiles = std::max(0LL, (long long)p->n_tiles - cost[2 * (size_t)p->n_k + j]);
            Load top = bins.top();
            bins.pop();
            items[top.second].push_back(j);
            bins.push(Load(top.first + cost[j] + per_tile * tiles + per_row, top.second));
        }
        std::vector<int32_t> bin_start(p->n_bins + 1, 0), bin_items;
        for (int b = 0; b < p->n_bins; ++b) {
            bin_items.insert(bin_items.end(), items[b].begin(), items[b].end());
            bin_start[b + 1] = (int32_t)bin_items.size();
        }
        GCAMB_CUDA(cudaMalloc(&p->d_bin_start, sizeof(int32_t) * bin_start.size()));
        GCAMB_CUDA(cudaMalloc(&p->d_bin_items, sizeof(int32_t) * p->n_k));
        GCAMB_CUDA(cudaMemcpyAsync(p->d_bin_start, bin_start.data(), sizeof(int32_t) * bin_start.size(), cudaMemcpyHostToDevice, stream));
        GCAMB_CUDA(cudaMemcpyAsync(p->d_bin_items, bin_items.data(), sizeof(int32_t) * p->n_k, cudaMemcpyHostToDevice, stream));
        GCAMB_CUDA(cudaStreamSynchronize(stream));   // the vectors die with this scope
    }
    // rows whose largest x = k chi_max exceeds COMP_X_MIN run the compensated coefficient; they
    // must be a prefix of the cost order (they are whenever cost grows with k), else all rows do
    {
        std::vector<double> hk(p->n_k);
        double chi_max = 0.0;
        GCAMB_CUDA(cudaMemcpyAsync(hk.data(), p->d_k, sizeof(double) * p->n_k, cudaMemcpyDeviceToHost, stream));
        GCAMB_CUDA(cudaMemcpyAsync(&chi_max, p->d_chi, sizeof(double), cudaMemcpyDeviceToHost, stream));   // tau grows: chi_0 is the largest
        GCAMB_CUDA(cudaStreamSynchronize(stream));
        int n_comp = 0;
        for (int j = 0; j < p->n_k; ++j) n_comp += hk[j] * chi_max > COMP_X_MIN;
        bool prefix = true;
        for (int r = 0; r < p->n_k; ++r) prefix = prefix && ((hk[order[r]] * chi_max > COMP_X_MIN) == (r < n_comp));
        p->n_comp = p->curved ? 0 : (prefix ? n_comp : p->n_k);   // the open-universe kernels have no compensated form
    }
    // zero region of Delta (R16): x grows with k, so the first tile of a k (that of tau_0, its
    // largest x) never rises with k, and the rows of tile t are exactly zero for the first kz[t]
    // k: the transfer kernel zeroes those row prefixes with coalesced stores.  The first tiles are
    // monotone for any valid (strictly increasing) k grid because L(x) is monotone in x; anything
    // else is an internal error and is reported, not worked around.
    const long long *first = cost.data() + 2 * (size_t)p->n_k;
    for (int j = 1; j < p->n_k; ++j) {
        if (first[j] > first[j - 1]) {
            set_error("internal: first l-tile not monotone in k at k index %d", j);
            return GCAMB_EGRID;
        }
    }
    std::vector<int32_t> kz(p->n_tiles);
    int j = p->n_k;   // kz[t] = #{k : first[k] > t}, non-increasing in t
    for (int t = 0; t < p->n_tiles; ++t) {
        while (j > 0 && first[j - 1] <= t) --j;
        kz[t] = j;
    }
    GCAMB_CUDA(cudaMalloc(&p->d_kz, sizeof(int32_t) * p->n_tiles));
    GCAMB_CUDA(cudaMemcpyAsync(p->d_kz, kz.data(), sizeof(int32_t) * p->n_tiles, cudaMemcpyHostToDevice, stream));
    GCAMB_CUDA(cudaStreamSynchronize(stream));
    return GCAMB_OK;
}

}  // namespace gcamb
