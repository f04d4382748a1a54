// api.cu -- the extern "C" boundary (include/gcamb_los.h): validation, host-side plan tables,
// launches.  No step of the hot path runs on the host.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "los_internal.cuh"

namespace gcamb {

static thread_local char g_err[512] = "";

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

gcamb_status cuda_fail(cudaError_t e, const char *what)
{
    set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    return e == cudaErrorMemoryAllocation ? GCAMB_EALLOC : GCAMB_ECUDA;
}

template <class Tp>
static cudaError_t upload(Tp **dst, const std::vector<Tp> &src, cudaStream_t s)
{
    cudaError_t e = cudaMalloc(dst, sizeof(Tp) * src.size());
    if (e != cudaSuccess) return e;
    return cudaMemcpyAsync(*dst, src.data(), sizeof(Tp) * src.size(), cudaMemcpyHostToDevice, s);
}

// composite-trapezoid weights on a non-uniform grid (R2, R6)
static std::vector<double> trapezoid(const std::vector<double> &t)
{
    const size_t n = t.size();
    std::vector<double> w(n);
    w[0] = 0.5 * (t[1] - t[0]);
    for (size_t i = 1; i + 1 < n; ++i) w[i] = 0.5 * (t[i + 1] - t[i - 1]);
    w[n - 1] = 0.5 * (t[n - 1] - t[n - 2]);
    return w;
}

static void free_plan(gcamb_los_plan *p)
{
    if (!p) return;
    std::free(p->h_k);
    cudaFree(p->d_l_index); cudaFree(p->d_k); cudaFree(p->d_chi); cudaFree(p->d_w);
    cudaFree(p->d_dlnk); cudaFree(p->d_pref); cudaFree(p->d_start); cudaFree(p->d_tile); cudaFree(p->d_inv);
    cudaFree(p->d_korder); cudaFree(p->d_l_list); cudaFree(p->d_kz); cudaFree(p->d_tile_mask);
    cudaFree(p->d_bin_start); cudaFree(p->d_bin_items); cudaFree(p->d_fused_scratch);
    cudaFree(p->d_sp_mult); cudaFree(p->d_sp_inv_diag); cudaFree(p->d_sp_seg); cudaFree(p->d_l_user);
    cudaFree(p->d_sp_ainv); cudaFree(p->d_sp_aoff); cudaFree(p->d_sp_alo); cudaFree(p->d_sp_acnt);
    cudaFree(p->d_cth); cudaFree(p->d_s2); cudaFree(p->d_ib2); cudaFree(p->d_coef); cudaFree(p->d_l_end);
    cudaFree(p->d_t_posm); cudaFree(p->d_t_pos0); cudaFree(p->d_t_pos1); cudaFree(p->d_t_pos2);
    cudaFree(p->d_t_cE); cudaFree(p->d_t_cB); cudaFree(p->d_t_c3);
    for (int q = 0; q < 3; ++q) cudaFree(p->d_hS[q]);
    cudaFree(p->d_hP); cudaFree(p->d_hDelta); cudaFree(p->d_hCl);
    if (p->h_streams_ready) {
        cudaStreamDestroy(p->h_copy);
        cudaEventDestroy(p->h_start);
        for (int c = 0; c < 4; ++c) { cudaStreamDestroy(p->h_comp[c]); cudaEventDestroy(p->h_copied[c]); cudaEventDestroy(p->h_done[c]); }
    }
    delete p;
}

// a plan's tables live on the device that was current at its creation; so must the caller's buffers
static gcamb_status check_device(const gcamb_los_plan *p)
{
    int dev = -1;
    GCAMB_CUDA(cudaGetDevice(&dev));
    if (dev != p->device) {
        set_error("plan belongs to device %d but device %d is current", p->device, dev);
        return GCAMB_EINVAL;
    }
    return GCAMB_OK;
}

static gcamb_status check_call(const gcamb_los_plan *p, int n_batch, const double *S_T,
                               const double *S_E, const double *S_phi, const void *out)
{
    if (!p || !S_T || !S_E || !out) { set_error("null plan or buffer"); return GCAMB_EINVAL; }
    if (p->tensor) { set_error("tensor plan: use gcamb_los_transfer_tensor / gcamb_los_cls_tensor"); return GCAMB_EINVAL; }
    if (gcamb_status st = check_device(p)) return st;
    if (n_batch < 1 || n_batch > 65535) { set_error("n_batch must be in [1, 65535]"); return GCAMB_EINVAL; }
    if ((long long)p->n_k * n_batch > 0x7fffffffLL) {   // one CTA per (k, cosmology) along grid.x
        set_error("n_k * n_batch must be below 2^31");
        return GCAMB_EINVAL;
    }
    if ((p->n_src == 3) != (S_phi != nullptr)) {
        set_error("S_phi must be non-NULL exactly when the plan has GCAMB_SRC_PHI");
        return GCAMB_EINVAL;
    }
    return GCAMB_OK;
}

}  // namespace gcamb

using namespace gcamb;

extern "C" {

const char *gcamb_los_last_error(void) { return g_err; }

}  // extern "C"

// curv_K = 0: flat; curv_K < 0: open universe (reading R28)
static gcamb_status create_plan(gcamb_los_plan **out, const int32_t *l_list, int32_t n_l,
                                const double *k, int32_t n_k, const double *tau, int32_t n_tau,
                                double tau0, double curv_K, uint32_t src_mask, void *cuda_stream)
{
    if (out) *out = nullptr;
    if (!out || !l_list || !k || !tau) { set_error("null argument"); return GCAMB_EINVAL; }
    if (n_l < 1 || n_k < 2 || n_tau < 2) { set_error("need n_l >= 1, n_k >= 2, n_tau >= 2"); return GCAMB_EINVAL; }
    const bool curved = curv_K != 0.0;
    if (!std::isfinite(curv_K)) { set_error("curvature K must be finite"); return GCAMB_EINVAL; }
    const int sgn = curv_K < 0.0 ? +1 : -1;     // +1 open, -1 closed
    const bool tensor = src_mask == GCAMB_SRC_TENSOR;
    if (curved && tensor) { set_error("tensor plans are flat only"); return GCAMB_EINVAL; }
    if (!tensor && src_mask != (GCAMB_SRC_T | GCAMB_SRC_E) && src_mask != (GCAMB_SRC_T | GCAMB_SRC_E | GCAMB_SRC_PHI)) {
        set_error("src_mask must be T|E, T|E|PHI or TENSOR");
        return GCAMB_EINVAL;
    }
    const int l_top = tensor ? 65533 : 65535;   // a tensor plan also walks l + 1 and l + 2
    for (int i = 0; i < n_l; ++i) {
        if (l_list[i] < 2 || l_list[i] > l_top) { set_error("l_list[%d] = %d outside [2, %d]", i, l_list[i], l_top); return GCAMB_EINVAL; }
        if (i && l_list[i] <= l_list[i - 1]) { set_error("l_list not strictly increasing at %d", i); return GCAMB_EINVAL; }
    }
    // Tensor plans (tensor.cu): every tensor transfer function is a combination of PLAIN sums at l - 1 .. l + 2, so
    // the kernels run on the union of those lists (l - 1 may be 1); the caller's list and the rows of l - 1 .. l + 2
    // in the union are kept.
    const int32_t *user_list = l_list;
    const int32_t n_user = n_l;
    std::vector<int32_t> ext, posm, pos0, pos1, pos2;
    if (tensor) {
        for (int i = 0; i < n_l; ++i)
            for (int d = -1; d <= 2; ++d) ext.push_back(l_list[i] + d);
        std::sort(ext.begin(), ext.end());
        ext.erase(std::unique(ext.begin(), ext.end()), ext.end());
        auto row_of = [&](int l) { return (int32_t)(std::lower_bound(ext.begin(), ext.end(), l) - ext.begin()); };
        for (int i = 0; i < n_l; ++i) {
            posm.push_back(row_of(l_list[i] - 1)); pos0.push_back(row_of(l_list[i]));
            pos1.push_back(row_of(l_list[i] + 1)); pos2.push_back(row_of(l_list[i] + 2));
        }
        l_list = ext.data();
        n_l = (int32_t)ext.size();
    }
    if (!std::isfinite(tau0)) { set_error("tau0 not finite"); return GCAMB_EGRID; }
    for (int j = 0; j < n_k; ++j) {
        if (!std::isfinite(k[j]) || !(k[j] > 0.0)) { set_error("k[%d] must be finite and > 0", j); return GCAMB_EGRID; }
        if (j && !(k[j] > k[j - 1])) { set_error("k not strictly increasing at %d", j); return GCAMB_EGRID; }
    }
    for (int i = 0; i < n_tau; ++i) {
        if (!std::isfinite(tau[i]) || !(tau[i] < tau0)) { set_error("tau[%d] must be finite and < tau0 (x > 0, R18)", i); return GCAMB_EGRID; }
        if (i && !(tau[i] > tau[i - 1])) { set_error("tau not strictly increasing at %d", i); return GCAMB_EGRID; }
    }

    gcamb_los_plan *p = new (std::nothrow) gcamb_los_plan();
    if (!p) { set_error("out of host memory"); return GCAMB_EALLOC; }
    std::memset(p, 0, sizeof(*p));
    p->n_l = n_l; p->n_k = n_k; p->n_tau = n_tau;
    p->n_l_out = n_user;
    p->tensor = tensor;
    p->curved = curved ? sgn : 0;
    p->r_c = curved ? 1.0 / std::sqrt(std::fabs(curv_K)) : 0.0;
    p->src_mask = src_mask;
    p->n_src = (tensor || (src_mask & GCAMB_SRC_PHI)) ? 3 : 2;
    p->n_src_walk = tensor ? 2 : p->n_src;
    p->l_user_first = user_list[0]; p->l_user_last = user_list[n_user - 1];
    p->n_spec = p->n_src + 1;
    p->l_min = l_list[0]; p->l_max = l_list[n_l - 1];
    p->tau0 = tau0;
    p->h_k = (double *)std::malloc(sizeof(double) * n_k);
    if (!p->h_k) { set_error("out of host memory"); free_plan(p); return GCAMB_EALLOC; }
    std::memcpy(p->h_k, k, sizeof(double) * n_k);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaGetDevice(&p->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, p->device);
    if (e != cudaSuccess) { gcamb_status st = cuda_fail(e, "device query"); free_plan(p); return st; }
    p->shape = choose_shape(n_tau, p->n_src_walk, n_k, p->n_sm);
    p->n_tiles = (p->l_max - p->l_min) / p->shape.V + 1;

    // IntegrationVars_init: the O(N) tables, on the host in fp64
    std::vector<double> vk(k, k + n_k), vtau(tau, tau + n_tau), chi(n_tau), lnk(n_k), pref(n_l);
    for (int i = 0; i < n_tau; ++i) chi[i] = tau0 - tau[i];
    std::vector<double> cth, s2, ib2;
    if (curved) {   // chi_i = sqrt|K| (tau0 - tau_i), one rounding, like the flat x = k chi; beta_j = k_j r_c
        const double sk = std::sqrt(std::fabs(curv_K));
        cth.resize(n_tau); s2.resize(n_tau); ib2.resize(n_k);
        for (int i = 0; i < n_tau; ++i) {
            chi[i] = sk * (tau0 - tau[i]);
            const double sh = sgn > 0 ? std::sinh(chi[i]) : std::sin(chi[i]);
            cth[i] = (sgn > 0 ? std::cosh(chi[i]) : std::cos(chi[i])) / sh;
            s2[i] = 1.0 / (sh * sh);
        }
        if (sgn < 0 && !(chi[0] <= 1.5707963267948966)) {
            set_error("closed universe: chi = sqrt(K) (tau0 - tau) must not exceed pi/2 (it is %.4f at tau[0])", chi[0]);
            free_plan(p);
            return GCAMB_EGRID;
        }
        for (int j = 0; j < n_k; ++j) {
            double beta = k[j] * p->r_c;
            if (sgn < 0) {   // closed: the modes are beta = 3, 4, 5, ...
                const double br = std::floor(beta + 0.5);
                if (br < 3.0 || std::fabs(beta - br) > 1e-6 * br) {
                    set_error("closed universe: k[%d] / sqrt(K) = %.9g is not an integer >= 3", j, beta);
                    free_plan(p);
                    return GCAMB_EGRID;
                }
                beta = br;
            }
            ib2[j] = 1.0 / (beta * beta);
        }
    }
    for (int j = 0; j < n_k; ++j) lnk[j] = std::log(k[j]);
    std::vector<double> w = trapezoid(vtau), dlnk = trapezoid(lnk);
    std::vector<int32_t> l_index((size_t)p->l_max + 1, -1);
    for (int i = 0; i < n_l; ++i) {
        const double l = l_list[i];
        l_index[l_list[i]] = i;
        pref[i] = std::sqrt((l + 2.0) * (l + 1.0) * l * (l - 1.0));   // (l+2)!/(l-2)!  (R3)
    }

    e = upload(&p->d_l_index, l_index, stream);
    if (e == cudaSuccess) e = upload(&p->d_l_list, std::vector<int32_t>(l_list, l_list + n_l), stream);
    if (e == cudaSuccess) e = upload(&p->d_l_user, std::vector<int32_t>(user_list, user_list + n_user), stream);
    if (tensor) {
        // combination coefficients of tensor.cu
        std::vector<double> cE(n_user), cB(n_user), c3(n_user);
        for (int i = 0; i < n_user; ++i) {
            const double l = user_list[i];
            cE[i] = (l + 1.0) * (l + 2.0) / std::sqrt((l + 2.0) * (l + 1.0) * l * (l - 1.0));
            cB[i] = 2.0 * (l + 2.0) / (2.0 * l + 1.0);
            c3[i] = 1.0 / (2.0 * l + 3.0);
        }
        if (e == cudaSuccess) e = upload(&p->d_t_posm, posm, stream);
        if (e == cudaSuccess) e = upload(&p->d_t_pos0, pos0, stream);
        if (e == cudaSuccess) e = upload(&p->d_t_pos1, pos1, stream);
        if (e == cudaSuccess) e = upload(&p->d_t_pos2, pos2, stream);
        if (e == cudaSuccess) e = upload(&p->d_t_cE, cE, stream);
        if (e == cudaSuccess) e = upload(&p->d_t_cB, cB, stream);
        if (e == cudaSuccess) e = upload(&p->d_t_c3, c3, stream);
    }
    {   // sparse l lists: which tiles hold a listed l (NULL table = all of them)
        std::vector<uint32_t> mask((p->n_tiles + 31) / 32, 0u);
        for (int i = 0; i < n_l; ++i) {
            const int t = (p->l_max - l_list[i]) / p->shape.V;
            mask[t >> 5] |= 1u << (t & 31);
        }
        int listed = 0;
        for (int t = 0; t < p->n_tiles; ++t) listed += (mask[t >> 5] >> (t & 31)) & 1u;
        if (listed < p->n_tiles && e == cudaSuccess) e = upload(&p->d_tile_mask, mask, stream);
    }
    if (e == cudaSuccess) e = upload(&p->d_k, vk, stream);
    if (e == cudaSuccess) e = upload(&p->d_chi, chi, stream);
    if (e == cudaSuccess) e = upload(&p->d_w, w, stream);
    if (e == cudaSuccess) e = upload(&p->d_dlnk, dlnk, stream);
    if (e == cudaSuccess) e = upload(&p->d_pref, pref, stream);
    const size_t npt = (size_t)n_k * n_tau;
    if (e == cudaSuccess) e = cudaMalloc(&p->d_start, sizeof(double2) * npt);
    if (e == cudaSuccess) e = cudaMalloc(&p->d_tile, sizeof(int32_t) * npt);
    if (e == cudaSuccess && !curved) e = cudaMalloc(&p->d_inv, sizeof(double) * npt);
    if (curved) {
        if (e == cudaSuccess) e = upload(&p->d_cth, cth, stream);
        if (e == cudaSuccess) e = upload(&p->d_s2, s2, stream);
        if (e == cudaSuccess) e = upload(&p->d_ib2, ib2, stream);
        if (e == cudaSuccess) e = cudaMalloc(&p->d_coef, sizeof(double2) * (size_t)n_k * p->n_tiles * p->shape.V);
        if (e == cudaSuccess) e = cudaMalloc(&p->d_l_end, sizeof(int32_t) * n_k);
    }
    if (e == cudaSuccess) e = cudaMalloc(&p->d_korder, sizeof(int32_t) * n_k);
    // the uploads read pageable vectors that die with this scope
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) { gcamb_status st = cuda_fail(e, "plan tables"); free_plan(p); return st; }

    gcamb_status st = plan_precompute(p, stream);
    if (st == GCAMB_OK) st = interp_plan_tables(p, user_list, stream);
    if (st != GCAMB_OK) { free_plan(p); return st; }
    *out = p;
    return GCAMB_OK;
}

extern "C" {

gcamb_status gcamb_los_plan_create(gcamb_los_plan **out, const int32_t *l_list, int32_t n_l,
                                   const double *k, int32_t n_k, const double *tau, int32_t n_tau,
                                   double tau0, uint32_t src_mask, void *cuda_stream)
{
    return create_plan(out, l_list, n_l, k, n_k, tau, n_tau, tau0, 0.0, src_mask, cuda_stream);
}

gcamb_status gcamb_los_plan_create_curved(gcamb_los_plan **out, const int32_t *l_list, int32_t n_l,
                                          const double *k, int32_t n_k, const double *tau, int32_t n_tau,
                                          double tau0, double curvature_K, uint32_t src_mask, void *cuda_stream)
{
    if (!(curvature_K != 0.0)) {
        if (out) *out = nullptr;
        set_error("gcamb_los_plan_create_curved needs K != 0 (K = 0: gcamb_los_plan_create)");
        return GCAMB_EINVAL;
    }
    return create_plan(out, l_list, n_l, k, n_k, tau, n_tau, tau0, curvature_K, src_mask, cuda_stream);
}

gcamb_status gcamb_los_plan_destroy(gcamb_los_plan *plan)
{
    if (!plan) return GCAMB_OK;
    // synchronise and free on the owning device, whatever device is current; restore the caller's
    int cur = -1;
    const int owner = plan->device;
    cudaError_t e = cudaGetDevice(&cur);
    if (e == cudaSuccess && cur != owner) e = cudaSetDevice(owner);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    free_plan(plan);
    if (cur >= 0 && cur != owner) cudaSetDevice(cur);
    if (e != cudaSuccess) return cuda_fail(e, "cudaDeviceSynchronize");
    return GCAMB_OK;
}

gcamb_status gcamb_los_plan_info(const gcamb_los_plan *plan, int32_t *n_l, int32_t *n_k, int32_t *n_tau,
                                 int32_t *n_src, int32_t *n_spec, int64_t *executed_terms)
{
    if (!plan) { set_error("null plan"); return GCAMB_EINVAL; }
    if (n_l) *n_l = plan->n_l_out;
    if (n_k) *n_k = plan->n_k;
    if (n_tau) *n_tau = plan->n_tau;
    if (n_src) *n_src = plan->n_src;
    if (n_spec) *n_spec = plan->n_spec;
    if (executed_terms) *executed_terms = plan->executed_terms;
    return GCAMB_OK;
}

gcamb_status gcamb_los_plan_launches(const gcamb_los_plan *plan, int32_t *transfer_kernels, int32_t *cls_kernels)
{
    if (!plan) { set_error("null plan"); return GCAMB_EINVAL; }
    if (transfer_kernels) *transfer_kernels = (plan->n_comp > 0) + (plan->n_comp < plan->n_k);
    if (cls_kernels) *cls_kernels = 1;
    return GCAMB_OK;
}

gcamb_status gcamb_los_transfer_batched(const gcamb_los_plan *plan, int32_t n_batch, const double *d_S_T,
                                        const double *d_S_E, const double *d_S_phi, double *d_Delta,
                                        void *cuda_stream)
{
    gcamb_status st = check_call(plan, n_batch, d_S_T, d_S_E, d_S_phi, d_Delta);
    if (st != GCAMB_OK) return st;
    return launch_transfer(plan, n_batch, d_S_T, d_S_E, d_S_phi, d_Delta, (cudaStream_t)cuda_stream);
}

gcamb_status gcamb_los_transfer(const gcamb_los_plan *plan, const double *d_S_T, const double *d_S_E,
                                const double *d_S_phi, double *d_Delta, void *cuda_stream)
{
    return gcamb_los_transfer_batched(plan, 1, d_S_T, d_S_E, d_S_phi, d_Delta, cuda_stream);
}

gcamb_status gcamb_los_cls_batched(const gcamb_los_plan *plan, int32_t n_batch, const double *d_Delta,
                                   const double *d_P_R, double *d_Cl, void *cuda_stream)
{
    if (!plan || !d_Delta || !d_P_R || !d_Cl) { set_error("null plan or buffer"); return GCAMB_EINVAL; }
    if (plan->tensor) { set_error("tensor plan: use gcamb_los_cls_tensor"); return GCAMB_EINVAL; }
    if (n_batch < 1 || n_batch > 65535) { set_error("n_batch must be in [1, 65535]"); return GCAMB_EINVAL; }
    if (gcamb_status st = check_device(plan)) return st;
    return launch_cls(plan, n_batch, d_Delta, d_P_R, d_Cl, (cudaStream_t)cuda_stream);
}

gcamb_status gcamb_los_cls(const gcamb_los_plan *plan, const double *d_Delta, const double *d_P_R,
                           double *d_Cl, void *cuda_stream)
{
    return gcamb_los_cls_batched(plan, 1, d_Delta, d_P_R, d_Cl, cuda_stream);
}

gcamb_status gcamb_los_tensor_work_bytes(const gcamb_los_plan *plan, int64_t *bytes)
{
    if (!plan || !bytes) { set_error("null argument"); return GCAMB_EINVAL; }
    if (!plan->tensor) { set_error("not a tensor plan"); return GCAMB_EINVAL; }
    *bytes = (int64_t)tensor_work_bytes(plan);
    return GCAMB_OK;
}

gcamb_status gcamb_los_transfer_tensor_batched(const gcamb_los_plan *plan, int32_t n_batch, const double *d_S_T,
                                               const double *d_S_E, const double *d_S_B, double *d_Delta,
                                               double *d_work, void *cuda_stream)
{
    if (!plan || !d_S_T || !d_S_E || !d_S_B || !d_Delta || !d_work) { set_error("null plan or buffer"); return GCAMB_EINVAL; }
    if (!plan->tensor) { set_error("not a tensor plan (create it with GCAMB_SRC_TENSOR)"); return GCAMB_EINVAL; }
    if (n_batch < 1 || n_batch > 32767) { set_error("n_batch must be in [1, 32767] for tensor plans"); return GCAMB_EINVAL; }
    if (2LL * plan->n_k * n_batch > 0x7fffffffLL) {   // one CTA per (k, run, cosmology) along grid.x
        set_error("2 * n_k * n_batch must be below 2^31");
        return GCAMB_EINVAL;
    }
    if (gcamb_status st = check_device(plan)) return st;
    return launch_transfer_tensor(plan, n_batch, d_S_T, d_S_E, d_S_B, d_Delta, d_work, (cudaStream_t)cuda_stream);
}

gcamb_status gcamb_los_transfer_tensor(const gcamb_los_plan *plan, const double *d_S_T, const double *d_S_E,
                                       const double *d_S_B, double *d_Delta, double *d_work, void *cuda_stream)
{
    return gcamb_los_transfer_tensor_batched(plan, 1, d_S_T, d_S_E, d_S_B, d_Delta, d_work, cuda_stream);
}

gcamb_status gcamb_los_cls_tensor_batched(const gcamb_los_plan *plan, int32_t n_batch, const double *d_Delta,
                                          const double *d_P_t, double *d_Cl, void *cuda_stream)
{
    if (!plan || !d_Delta || !d_P_t || !d_Cl) { set_error("null plan or buffer"); return GCAMB_EINVAL; }
    if (!plan->tensor) { set_error("not a tensor plan (create it with GCAMB_SRC_TENSOR)"); return GCAMB_EINVAL; }
    if (n_batch < 1 || n_batch > 65535) { set_error("n_batch must be in [1, 65535]"); return GCAMB_EINVAL; }
    if (gcamb_status st = check_device(plan)) return st;
    // Eq. 1 on (T, E, B): the scalar kernels' (TT, EE, TE, third-source auto) written in the order TT, EE, BB, TE
    return launch_cls(plan, n_batch, d_Delta, d_P_t, d_Cl, (cudaStream_t)cuda_stream);
}

gcamb_status gcamb_los_cls_tensor(const gcamb_los_plan *plan, const double *d_Delta, const double *d_P_t,
                                  double *d_Cl, void *cuda_stream)
{
    return gcamb_los_cls_tensor_batched(plan, 1, d_Delta, d_P_t, d_Cl, cuda_stream);
}

gcamb_status gcamb_los_cl_interp(const gcamb_los_plan *plan, int32_t n_batch, const double *d_Cl,
                                 double *d_Cl_all, void *cuda_stream)
{
    if (!plan || !d_Cl || !d_Cl_all) { set_error("null plan or buffer"); return GCAMB_EINVAL; }
    if (n_batch < 1 || n_batch > 65535) { set_error("n_batch must be in [1, 65535]"); return GCAMB_EINVAL; }
    if (gcamb_status st = check_device(plan)) return st;
    return launch_cl_interp(plan, n_batch, d_Cl, d_Cl_all, (cudaStream_t)cuda_stream);
}

gcamb_status gcamb_los_spectra_batched(gcamb_los_plan *plan, int32_t n_batch, const double *d_S_T,
                                       const double *d_S_E, const double *d_S_phi, const double *d_P_R,
                                       double *d_Cl, void *cuda_stream)
{
    gcamb_status st = check_call(plan, n_batch, d_S_T, d_S_E, d_S_phi, d_Cl);
    if (st != GCAMB_OK) return st;
    if (!d_P_R) { set_error("null P_R"); return GCAMB_EINVAL; }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const bool fused = fused_supported(plan, n_batch);
    // scratch: the fused kernel's partial spectra, else the Delta of the two-kernel path
    const size_t need = fused ? fused_scratch_bytes(plan, n_batch)
                              : sizeof(double) * (size_t)n_batch * plan->n_src * plan->n_l * plan->n_k;
    if (need > plan->fused_scratch_cap) {
        // grow-only; a buffer still in use by earlier work on another stream must not be freed under it
        GCAMB_CUDA(cudaDeviceSynchronize());
        cudaFree(plan->d_fused_scratch);
        plan->d_fused_scratch = nullptr;
        plan->fused_scratch_cap = 0;
        GCAMB_CUDA(cudaMalloc(&plan->d_fused_scratch, need));
        plan->fused_scratch_cap = need;
    }
    if (fused) return launch_fused(plan, n_batch, d_S_T, d_S_E, d_P_R, plan->d_fused_scratch, d_Cl, s);
    st = launch_transfer(plan, n_batch, d_S_T, d_S_E, d_S_phi, plan->d_fused_scratch, s);
    if (st != GCAMB_OK) return st;
    return launch_cls(plan, n_batch, plan->d_fused_scratch, d_P_R, d_Cl, s);
}

gcamb_status gcamb_los_spectra_batched_info(const gcamb_los_plan *plan, int32_t n_batch, int32_t *fused,
                                            int32_t *kernels, int64_t *scratch_bytes)
{
    if (!plan || n_batch < 1) { set_error("null plan or n_batch < 1"); return GCAMB_EINVAL; }
    const bool f = fused_supported(plan, n_batch);
    if (fused) *fused = f;
    if (kernels) *kernels = f ? 2 : (plan->n_comp > 0) + (plan->n_comp < plan->n_k) + 1;
    if (scratch_bytes)
        *scratch_bytes = (int64_t)(f ? fused_scratch_bytes(plan, n_batch)
                                     : sizeof(double) * (size_t)n_batch * plan->n_src * plan->n_l * plan->n_k);
    return GCAMB_OK;
}

}  // extern "C"

constexpr size_t HOST_PIPELINE_MIN_BYTES = 4u << 20;

// everything gcamb_los_spectra_host enqueues; on an error the caller joins the streams before returning
static gcamb_status spectra_host_enqueue(gcamb_los_plan *p, int32_t n_batch, const double *h_S_T,
                                         const double *h_S_E, const double *h_S_phi, const double *h_P_R,
                                         double *h_Cl, double *h_Delta, cudaStream_t s)
{
    gcamb_status st;
    const size_t nS = (size_t)p->n_k * p->n_tau, nD = (size_t)p->n_src * p->n_l * p->n_k;
    const size_t nC = (size_t)p->n_spec * p->n_l;
    if (n_batch > p->host_batch_cap) {
        for (int q = 0; q < 3; ++q) { cudaFree(p->d_hS[q]); p->d_hS[q] = nullptr; }
        cudaFree(p->d_hP); cudaFree(p->d_hDelta); cudaFree(p->d_hCl);
        p->d_hP = p->d_hDelta = p->d_hCl = nullptr;
        p->host_batch_cap = 0;
        for (int q = 0; q < p->n_src; ++q) GCAMB_CUDA(cudaMalloc(&p->d_hS[q], sizeof(double) * nS * n_batch));
        GCAMB_CUDA(cudaMalloc(&p->d_hP, sizeof(double) * p->n_k * n_batch));
        GCAMB_CUDA(cudaMalloc(&p->d_hDelta, sizeof(double) * nD * n_batch));
        GCAMB_CUDA(cudaMalloc(&p->d_hCl, sizeof(double) * nC * n_batch));
        p->host_batch_cap = n_batch;
    }
    const double *hS[3] = {h_S_T, h_S_E, h_S_phi};
    GCAMB_CUDA(cudaMemcpyAsync(p->d_hP, h_P_R, sizeof(double) * p->n_k * n_batch, cudaMemcpyHostToDevice, s));

    // The rows are processed heaviest first = k descending, so a range of cost-order positions is a
    // contiguous block of k rows: the sources go up in NCH blocks on a copy stream and each block's
    // kernels start on a stream of their own as soon as it has landed.  The first block is small
    // (little to wait for, and its rows carry a third of the work), the last one is half the rows
    // (light ones).  H2D of 8 n_src N_k N_tau bytes bounds the call; compute hides behind it.
    constexpr int NCH = 4;
    // (below HOST_PIPELINE_MIN_BYTES of sources the ~40 stream and event calls of the pipeline cost more than
    // the overlap returns: config 0, 1.9 MB, 136 us pipelined)
    const bool pipelined = p->order_reversed && p->n_k >= 64 &&
                           sizeof(double) * nS * n_batch * p->n_src >= HOST_PIPELINE_MIN_BYTES;
    if (pipelined && !p->h_streams_ready) {
        GCAMB_CUDA(cudaStreamCreateWithFlags(&p->h_copy, cudaStreamNonBlocking));
        GCAMB_CUDA(cudaEventCreateWithFlags(&p->h_start, cudaEventDisableTiming));
        for (int c = 0; c < NCH; ++c) {
            GCAMB_CUDA(cudaStreamCreateWithFlags(&p->h_comp[c], cudaStreamNonBlocking));
            GCAMB_CUDA(cudaEventCreateWithFlags(&p->h_copied[c], cudaEventDisableTiming));
            GCAMB_CUDA(cudaEventCreateWithFlags(&p->h_done[c], cudaEventDisableTiming));
        }
        p->h_streams_ready = 1;
    }
    if (!pipelined) {
        for (int q = 0; q < p->n_src; ++q)
            GCAMB_CUDA(cudaMemcpyAsync(p->d_hS[q], hS[q], sizeof(double) * nS * n_batch, cudaMemcpyHostToDevice, s));
        st = launch_transfer_range(p, n_batch, p->d_hS[0], p->d_hS[1], p->d_hS[2], p->d_hDelta, 0, p->n_k, true, s);
        if (st != GCAMB_OK) return st;
    } else {
        const int bound[NCH + 1] = {0, p->n_k / 16, p->n_k / 4, p->n_k / 2, p->n_k};
        GCAMB_CUDA(cudaEventRecord(p->h_start, s));               // everything below follows the caller's stream
        GCAMB_CUDA(cudaStreamWaitEvent(p->h_copy, p->h_start, 0));
        const size_t pitch = sizeof(double) * nS;                  // one cosmology's [n_k][n_tau]
        for (int c = 0; c < NCH; ++c) {
            const int k_lo = p->n_k - bound[c + 1], rows = bound[c + 1] - bound[c];   // positions -> k rows
            const size_t off = (size_t)k_lo * p->n_tau;
            for (int q = 0; q < p->n_src; ++q)
                GCAMB_CUDA(cudaMemcpy2DAsync(p->d_hS[q] + off, pitch, hS[q] + off, pitch,
                                             sizeof(double) * (size_t)rows * p->n_tau, (size_t)n_batch,
                                             cudaMemcpyHostToDevice, p->h_copy));
            GCAMB_CUDA(cudaEventRecord(p->h_copied[c], p->h_copy));
            GCAMB_CUDA(cudaStreamWaitEvent(p->h_comp[c], p->h_start, 0));
            GCAMB_CUDA(cudaStreamWaitEvent(p->h_comp[c], p->h_copied[c], 0));
            st = launch_transfer_range(p, n_batch, p->d_hS[0], p->d_hS[1], p->d_hS[2], p->d_hDelta,
                                       bound[c], bound[c + 1], c == NCH - 1, p->h_comp[c]);
            if (st != GCAMB_OK) return st;
            GCAMB_CUDA(cudaEventRecord(p->h_done[c], p->h_comp[c]));
            GCAMB_CUDA(cudaStreamWaitEvent(s, p->h_done[c], 0));
        }
    }
    st = launch_cls(p, n_batch, p->d_hDelta, p->d_hP, p->d_hCl, s);
    if (st != GCAMB_OK) return st;
    GCAMB_CUDA(cudaMemcpyAsync(h_Cl, p->d_hCl, sizeof(double) * nC * n_batch, cudaMemcpyDeviceToHost, s));
    if (h_Delta)
        GCAMB_CUDA(cudaMemcpyAsync(h_Delta, p->d_hDelta, sizeof(double) * nD * n_batch, cudaMemcpyDeviceToHost, s));
    return GCAMB_OK;
}

extern "C" {

gcamb_status gcamb_los_spectra_host(gcamb_los_plan *plan, int32_t n_batch, const double *h_S_T,
                                    const double *h_S_E, const double *h_S_phi, const double *h_P_R,
                                    double *h_Cl, double *h_Delta, void *cuda_stream)
{
    gcamb_status st = check_call(plan, n_batch, h_S_T, h_S_E, h_S_phi, h_Cl);
    if (st != GCAMB_OK) return st;
    if (!h_P_R) { set_error("null P_R"); return GCAMB_EINVAL; }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    st = spectra_host_enqueue(plan, n_batch, h_S_T, h_S_E, h_S_phi, h_P_R, h_Cl, h_Delta, s);
    // Join every stream the call may have used, also on the error path: asynchronous copies from and to
    // the caller's buffers must not be in flight when the call returns.
    cudaError_t e = cudaStreamSynchronize(s);
    if (plan->h_streams_ready) {
        cudaError_t e2 = cudaStreamSynchronize(plan->h_copy);
        if (e == cudaSuccess) e = e2;
        for (int c = 0; c < 4; ++c) {
            e2 = cudaStreamSynchronize(plan->h_comp[c]);
            if (e == cudaSuccess) e = e2;
        }
    }
    if (st != GCAMB_OK) return st;
    if (e != cudaSuccess) return cuda_fail(e, "gcamb_los_spectra_host: stream synchronisation");
    return GCAMB_OK;
}

}  // extern "C"

