// Internal declarations shared by the translation units of libgcamb_los.so.
// Nothing here is visible through the C ABI (include/gcamb_los.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "gcamb_los.h"

namespace gcamb {

// Geometry of the transfer kernel chosen at plan creation.
struct TransferShape {
    int V;        // l-tile: accumulators per source per thread, = granularity of start tiles
    int T;        // (k, tau) points ("slots") carried per thread
    int threads;  // CTA size (multiple of 32)
    int n_pass;   // passes of one CTA over the tau range (n_tau > threads * T: pass p adds to passes < p)
    int pass_len; // tau points per pass (the last pass may be shorter)
};

}  // namespace gcamb

struct gcamb_los_plan {
    int32_t n_l, n_k, n_tau, n_src, n_spec, l_min, l_max, n_tiles;
    int32_t n_l_out;         // multipoles of the caller's list (= n_l, except for tensor plans: n_l counts l - 1 .. l + 2)
    int32_t l_user_first, l_user_last;   // first and last multipole of the caller's list
    int32_t n_src_walk;      // sources of the transfer kernels (= n_src, except for tensor plans: their shape is that of the two-source kernels, the call runs the four-sum ones)
    int32_t tensor;          // tensor-mode plan (tensor.cu)
    int32_t curved;          // 0 flat; +1 open, -1 closed universe (reading R28): hyperspherical Bessel functions
    double r_c;              // curvature radius 1/sqrt(-K) (curved plans)
    uint32_t src_mask;
    double tau0;
    gcamb::TransferShape shape;
    int64_t executed_terms;  // sum over (k,tau) of #l in [l_min, min(L(x), l_max)]
    int32_t n_comp;          // leading positions of korder that run the compensated coefficient (transfer.cu)
    int64_t walked_terms;    // same with the tile-aligned start the kernel really walks
    int device;              // the device that owns the tables; every call checks it is the current one
    int n_sm;                // its SM count

    double *h_k;             // HOST copy of the k grid [n_k] (srcinterp.cu builds its tables from it)

    // device tables
    int32_t *d_l_index;  // [l_max+1] position in l_list, or -1
    double *d_k;         // [n_k]
    double *d_chi;       // [n_tau] tau0 - tau_i
    double *d_w;         // [n_tau] trapezoid weights
    double *d_dlnk;      // [n_k]   trapezoid weights of ln k
    double *d_pref;      // [n_l]   sqrt((l+2)(l+1)l(l-1))
    double2 *d_start;    // [n_k][n_tau] (j_{lhi+1}(x), j_{lhi}(x)), lhi = l_max - V*tile
    int32_t *d_tile;     // [n_k][n_tau] first l-tile of the point
    double *d_inv;       // [n_k][n_tau] 1/x
    int32_t *d_korder;   // [n_k] k indices, heaviest first
    int32_t *d_l_list;   // [n_l] the l list
    uint32_t *d_tile_mask;   // [ceil(n_tiles/32)] bit t%32 of word t/32: tile t holds a listed l; NULL when every tile does
    int32_t *d_kz;       // [n_tiles] #k whose walk starts below tile t: Delta rows of tile t are 0 for k < kz[t]

    int32_t order_reversed;  // korder[r] == n_k - 1 - r: a range of positions is a contiguous range of k

    // fused batched path (fused.cu): static, cost-balanced lists of k rows, one per thread block slot
    int32_t n_bins;          // = n_sm
    int32_t *d_bin_start;    // [n_bins + 1]
    int32_t *d_bin_items;    // [n_k] k indices grouped by bin, heaviest first inside a bin
    // scratch of gcamb_los_spectra_batched (lazily allocated, grow-only)
    double *d_fused_scratch;
    size_t fused_scratch_cap;   // bytes

    // interpolation in l (interp.cu, reading R25): LU factors of the natural-spline system of the l list
    double *d_sp_mult;       // [n_l] forward-elimination multipliers
    double *d_sp_inv_diag;   // [n_l] reciprocals of the eliminated diagonal
    int32_t *d_sp_seg;       // [l_max - l_min + 1] knot interval of every integer l
    double *d_sp_ainv;       // banded inverse of the spline matrix, packed rows (interp.cu); NULL: the sequential sweeps are used
    int32_t *d_sp_aoff, *d_sp_alo, *d_sp_acnt;   // [n_l] offset, first column and number of columns of row i
    int32_t *d_l_user;       // [n_l_out] the caller's l list (knots of the spline)

    // open-universe plans: d_chi holds chi_i = (tau0 - tau_i)/r_c; d_inv is not allocated
    double *d_cth;           // [n_tau] coth(chi_i)
    double *d_s2;            // [n_tau] 1/sinh^2(chi_i)
    double *d_ib2;           // [n_k]   1/beta_j^2, beta_j = k_j r_c
    double2 *d_coef;         // [n_k][n_tiles V] (A_l, R_l) = ((2l+1)/b_l, b_{l+1}/b_l), l = l_max - index
    int32_t *d_l_end;        // [n_k]   closed: beta - 1, the last l with a non-zero function; open: INT_MAX

    // tensor plans: positions of l and l + 1 of the caller's list in l_list, combination coefficients
    int32_t *d_t_posm, *d_t_pos0, *d_t_pos1, *d_t_pos2;   // [n_l_out] rows of l - 1, l, l + 1, l + 2 in the kernels' list
    double *d_t_cE, *d_t_cB, *d_t_c3;   // [n_l_out] (l+1)(l+2)/sqrt((l+2)(l+1)l(l-1)),  2(l+2)/(2l+1),  1/(2l+3)

    // scratch of gcamb_los_spectra_host (lazily allocated)
    cudaStream_t h_copy, h_comp[4];
    cudaEvent_t h_start, h_copied[4], h_done[4];
    int32_t h_streams_ready;
    int32_t host_batch_cap;
    double *d_hS[3], *d_hP, *d_hDelta, *d_hCl;
};

namespace gcamb {

void set_error(const char *fmt, ...);
gcamb_status cuda_fail(cudaError_t e, const char *what);

#define GCAMB_CUDA(call)                                                   \
    do {                                                                   \
        cudaError_t e__ = (call);                                          \
        if (e__ != cudaSuccess) return ::gcamb::cuda_fail(e__, #call);     \
    } while (0)

// plan.cu: fills d_start / d_tile / d_korder / executed_terms on `stream` (synchronises it).
gcamb_status plan_precompute(gcamb_los_plan *p, cudaStream_t stream);

// transfer.cu
// x above which the systematic phase error x 2^-53 of the rounded reciprocal exceeds 7.5e-13 rad
//
constexpr double COMP_X_MIN = 6755.399441055744;   // 2^53 * 7.5e-13
int transfer_tile_v();
// n_rows = the k rows of ONE cosmology (a batched call must take the shape of the single call)
TransferShape choose_shape(int n_tau, int n_src, long long n_rows, int n_sm);
gcamb_status launch_transfer(const gcamb_los_plan *p, int n_batch, const double *S_T,
                             const double *S_E, const double *S_phi, double *Delta,
                             cudaStream_t stream);
// the same in pieces, for the pipelined host entry point: any partition of the cost-order positions
// [0, n_k) into ranges, exactly one of them (any) with zero_fill (that range zeroes the skipped
// region of ALL rows)
gcamb_status launch_transfer_range(const gcamb_los_plan *p, int n_batch, const double *S_T,
                                   const double *S_E, const double *S_phi, double *Delta,
                                   int pos0, int pos1, bool zero_fill, cudaStream_t stream);

// four sums in one walk (tensor.cu): Delta [n_batch][4][n_l][n_k] = sums of S_0 and S_2 (plain), S_1 and S_3 (1/x^2,
// with the sqrt((l+2)!/(l-2)!) prefactor); flat plans only.  The few heaviest rows go out as 256-thread blocks in a launch
// of their own, overlapped by the launch of the others (transfer.cu)
gcamb_status launch_transfer4(const gcamb_los_plan *p, int n_batch, const double *S_0, const double *S_1,
                              const double *S_2, const double *S_3, double *Delta, cudaStream_t stream);

// fused.cu: sources of a batch -> C_l in one kernel (no Delta), for T+E plans whose tau grid fits
bool fused_supported(const gcamb_los_plan *p, int n_batch);
size_t fused_scratch_bytes(const gcamb_los_plan *p, int n_batch);
gcamb_status launch_fused(const gcamb_los_plan *p, int n_batch, const double *S_T, const double *S_E,
                          const double *P_R, double *scratch, double *Cl, cudaStream_t stream);

// interp.cu: C_l on every integer l of [l_min, l_max] from C_l on the l list (natural cubic spline of l(l+1) C_l)
constexpr size_t INTERP_SMEM_MAX = 200000;   // two doubles and an int per knot in shared memory: n_l <= 10000
gcamb_status interp_plan_tables(gcamb_los_plan *p, const int32_t *l_list, cudaStream_t stream);
gcamb_status launch_cl_interp(const gcamb_los_plan *p, int n_batch, const double *Cl_samp, double *Cl_all,
                              cudaStream_t stream);

// tensor.cu: tensor-mode transfer functions from one run of the four-sum transfer kernels
size_t tensor_work_bytes(const gcamb_los_plan *p);
gcamb_status launch_transfer_tensor(const gcamb_los_plan *p, int n_batch, const double *S_T, const double *S_E,
                                    const double *S_B, double *Delta, double *work, cudaStream_t stream);

// cls.cu (tensor plans: rows of n_l_out multipoles, spectra written in the order TT, EE, BB, TE)
gcamb_status launch_cls(const gcamb_los_plan *p, int n_batch, const double *Delta,
                        const double *P_R, double *Cl, cudaStream_t stream);

}  // namespace gcamb
