// tensor.cu -- tensor-mode transfer functions (the second SourceToTransfers call of
// PAPER.md:131 and Figure 1; reading R27: the flat-space tensor kernels of the line-of-sight
// literature the paper cites at PAPER.md:54 and PAPER.md:331):
//   Delta^{T,t}_l = sqrt((l+2)!/(l-2)!) sum_i w_i S_T j_l(x_i) / x_i^2
//   Delta^{E,t}_l = sum_i w_i S_E [ -j_l + j_l'' + 2 j_l / x^2 + 4 j_l' / x ](x_i)
//   Delta^{B,t}_l = sum_i w_i S_B [ 2 j_l' + 4 j_l / x ](x_i)
// With j_l' = (l/x) j_l - j_{l+1} and the defining equation for j_l'' the radial kernels are
//   E:  -2 j_l + (l+1)(l+2) j_l / x^2 - (2/x) j_{l+1}          B:  2 (l+2) j_l / x - 2 j_{l+1}
// i.e. every transfer function is a combination, with coefficients that depend on l only, of PLAIN sums
//   [S, p]_l = sum_i w_i S(k, tau_i) x_i^-p j_l(x_i),   p = 0, 1, 2.
// The p = 1 sums follow from the p = 0 sums of the neighbouring multipoles through the recurrence itself,
//   j_l(x) / x = (j_{l-1}(x) + j_{l+1}(x)) / (2l+1)   =>   [S, 1]_l = ([S, 0]_{l-1} + [S, 0]_{l+1}) / (2l+1),
// (above the turning point the two terms nearly cancel, the sum is smaller than either by l/x; but a p = 1 sum
// enters a transfer function only next to a p = 0 sum of full size, so what counts is its ABSOLUTE error, which
// is that of the p = 0 sums; the p = 2 sums are NOT taken that way: they stand alone in Delta^T, and applied
// twice the identity would lose (x/l)^2),
// so FOUR plain sums suffice:
//   U1 = [S_E, 0]   U2 = [S_E, 2]   V2 = [S_B, 0]   W = [S_T, 2]
//   Delta^T_l = pref_l W_l
//   Delta^E_l = -2 U1_l + (l+1)(l+2) U2_l - 2 (U1_l + U1_{l+2}) / (2l+3)
//   Delta^B_l = 2 (l+2) (V2_{l-1} + V2_{l+1}) / (2l+1) - 2 V2_{l+1}.
// A (p = 0, p = 2 with the sqrt((l+2)!/(l-2)!) prefactor) pair of sums is exactly what the scalar T, E transfer
// kernel computes (a2 + a3: recurrence in registers, tau-sum, reduction), so the tensor path is ONE run of the
// four-sum instantiation of transfer.cu (NSRC = 4: two such pairs in one walk) on a plan whose l list is the union
// of {l - 1, l, l + 1, l + 2}:
//   sources (S_E, S_E, S_B, S_T) -> rows (U1, pref U2, V2, pref W = Delta^T)
// read in place (no copy of the sources), with a small kernel behind that combines the rows: 6 FP64 instructions
// per executed (l, k, tau) term.  Earlier forms of this file: the three-source kernels run twice with S / x as
// third source (six sums, 10 instructions per term): 0.423 ms at the paper's tensor sizes; two runs of the
// two-source kernels as one batched launch behind a kernel that laid the sources out as that batch (8 instructions
// per term): 0.313 ms.  Now 0.259 ms, with the few heaviest rows in a launch of 256-thread blocks of their own that
// the launch of the others overlaps (launch_transfer4, transfer.cu).
#include <algorithm>

#include "los_internal.cuh"

namespace gcamb {

namespace {

// raw: [B][4][n_le][n_k] (rows of the union list; sums U1, pref U2, V2, pref W); Delta: [B][3][n_l][n_k] (rows of the caller's list)
__global__ void __launch_bounds__(256) tensor_combine_kernel(const double *__restrict__ raw,
                                                             const int32_t *__restrict__ posm, const int32_t *__restrict__ pos0,
                                                             const int32_t *__restrict__ pos1, const int32_t *__restrict__ pos2,
                                                             const double *__restrict__ cE, const double *__restrict__ cB,
                                                             const double *__restrict__ c3,
                                                             double *__restrict__ Delta, int n_l, int n_le, int n_k)
{
    const int a = blockIdx.y;
    const size_t rm = (size_t)posm[a] * n_k, r0 = (size_t)pos0[a] * n_k, r1 = (size_t)pos1[a] * n_k, r2 = (size_t)pos2[a] * n_k;
    const size_t plane = (size_t)n_le * n_k;
    const double *rawA = raw + (size_t)blockIdx.z * 4 * plane, *rawB = rawA + 2 * plane;
    const double ce = cE[a], cb = cB[a], c3a = c3[a];
    const size_t oplane = (size_t)n_l * n_k, out = (size_t)blockIdx.z * 3 * oplane + (size_t)a * n_k;
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_k; j += gridDim.x * blockDim.x) {
        const double U1 = rawA[r0 + j], U1pp = rawA[r2 + j], pU2 = rawA[plane + r0 + j];
        const double V2m = rawB[rm + j], V2p = rawB[r1 + j], pW = rawB[plane + r0 + j];
        Delta[out + j] = pW;
        Delta[oplane + out + j] = fma(ce, pU2, -2.0 * U1) - 2.0 * ((U1 + U1pp) * c3a);
        Delta[2 * oplane + out + j] = fma(cb, V2m + V2p, -2.0 * V2p);
    }
}

}  // namespace

size_t tensor_work_bytes(const gcamb_los_plan *p)
{
    return sizeof(double) * 4 * (size_t)p->n_l * p->n_k;
}

gcamb_status launch_transfer_tensor(const gcamb_los_plan *p, int n_batch, const double *S_T, const double *S_E,
                                    const double *S_B, double *Delta, double *work, cudaStream_t stream)
{
    double *raw = work;   // [B][4][n_le][n_k]
    gcamb_status st = launch_transfer4(p, n_batch, S_E, S_E, S_B, S_T, raw, stream);
    if (st != GCAMB_OK) return st;
    dim3 grid((unsigned)std::min((p->n_k + 255) / 256, 64), (unsigned)p->n_l_out, (unsigned)n_batch);
    tensor_combine_kernel<<<grid, 256, 0, stream>>>(raw, p->d_t_posm, p->d_t_pos0, p->d_t_pos1, p->d_t_pos2,
                                                    p->d_t_cE, p->d_t_cB, p->d_t_c3, Delta, p->n_l_out, p->n_l, p->n_k);
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

}  // namespace gcamb
