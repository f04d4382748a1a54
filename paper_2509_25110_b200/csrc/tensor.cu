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
// kernel computes (a2 + a3: recurrence in registers, tau-sum, reduction), so the tensor path is two runs of the
// TWO-source kernels of transfer.cu (the fast ones: three thread blocks per SM) on a plan whose l list is the
// union of {l - 1, l, l + 1, l + 2}:
//   run A: (S_E, S_E) -> (U1, pref U2)      run B: (S_B, S_T) -> (V2, pref W = Delta^T)
// issued as one batched launch of two members per cosmology, with a small kernel in front that lays the sources
// out as that batch and a small kernel behind that combines the rows.  8 FP64 instructions per executed (l, k, tau)
// term (a single walk with four sums would need 6).  The first form of this file ran the three-source kernels
// twice with S / x as third source (six sums, 10 instructions per term, two thread blocks per SM): 0.423 ms at the
// paper's tensor sizes against 0.28 ms now.
#include <algorithm>

#include "los_internal.cuh"

namespace gcamb {

namespace {

// The two runs go out as ONE batched launch (twice the thread blocks: a finer tail than two launches of n_k
// blocks each), so their sources are laid out as a batch of two per kernel slot and cosmology b:
//   slot 0 = [.. S_E(b) | S_B(b) ..]  (p = 0),   slot 1 = [.. S_E(b) | S_T(b) ..]  (p = 2, prefactor)
// member 2 b of the launch is run A of cosmology b, member 2 b + 1 its run B.
__global__ void __launch_bounds__(256) tensor_prep_kernel(const double *__restrict__ S_T, const double *__restrict__ S_E,
                                                          const double *__restrict__ S_B, double *__restrict__ slot0,
                                                          double *__restrict__ slot1, size_t n)
{
    const size_t in = (size_t)blockIdx.y * n, out = 2 * in;   // cosmology blockIdx.y
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double t = S_T[in + i], e = S_E[in + i], b = S_B[in + i];
        slot0[out + i] = e; slot0[out + n + i] = b;
        slot1[out + i] = e; slot1[out + n + i] = t;
    }
}

// raw: [B][2 runs][2][n_le][n_k] (rows of the union list); Delta: [B][3][n_l][n_k] (rows of the caller's list)
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
    return sizeof(double) * (4 * (size_t)p->n_k * p->n_tau + 4 * (size_t)p->n_l * p->n_k);
}

gcamb_status launch_transfer_tensor(const gcamb_los_plan *p, int n_batch, const double *S_T, const double *S_E,
                                    const double *S_B, double *Delta, double *work, cudaStream_t stream)
{
    const size_t n_pt = (size_t)p->n_k * p->n_tau, B = (size_t)n_batch;
    double *slot0 = work, *slot1 = work + 2 * B * n_pt, *raw = work + 4 * B * n_pt;
    const unsigned blocks = (unsigned)std::min<size_t>((n_pt + 255) / 256, (size_t)p->n_sm * 16);
    tensor_prep_kernel<<<dim3(blocks, (unsigned)n_batch), 256, 0, stream>>>(S_T, S_E, S_B, slot0, slot1, n_pt);
    GCAMB_CUDA(cudaGetLastError());
    // member 2 b = run A of cosmology b, member 2 b + 1 = its run B: raw [B][2][2][n_le][n_k]
    gcamb_status st = launch_transfer(p, 2 * n_batch, slot0, slot1, nullptr, raw, stream);
    if (st != GCAMB_OK) return st;
    dim3 grid((unsigned)std::min((p->n_k + 255) / 256, 64), (unsigned)p->n_l_out, (unsigned)n_batch);
    tensor_combine_kernel<<<grid, 256, 0, stream>>>(raw, p->d_t_posm, p->d_t_pos0, p->d_t_pos1, p->d_t_pos2,
                                                    p->d_t_cE, p->d_t_cB, p->d_t_c3, Delta, p->n_l_out, p->n_l, p->n_k);
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

}  // namespace gcamb
