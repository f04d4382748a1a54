// tensor.cu -- tensor-mode transfer functions (the second SourceToTransfers call of
// PAPER.md:131 and Figure 1; reading R27: the flat-space tensor kernels of the line-of-sight
// literature the paper cites at PAPER.md:54 and PAPER.md:331):
//   Delta^{T,t}_l = sqrt((l+2)!/(l-2)!) sum_i w_i S_T j_l(x_i) / x_i^2
//   Delta^{E,t}_l = sum_i w_i S_E [ -j_l + j_l'' + 2 j_l / x^2 + 4 j_l' / x ](x_i)
//   Delta^{B,t}_l = sum_i w_i S_B [ 2 j_l' + 4 j_l / x ](x_i)
// With j_l' = (l/x) j_l - j_{l+1} and the defining equation for j_l'' the radial kernels are
//   E:  -2 j_l + (l+1)(l+2) j_l / x^2 - (2/x) j_{l+1}          B:  2 (l+2) j_l / x - 2 j_{l+1}
// i.e. every transfer function is a combination, with coefficients that depend on l only, of PLAIN sums
//   sum_i w_i S(k, tau_i) x_i^-p j_l(x_i),   p = 0, 1, 2,   taken at l and at l + 1:
//   U1 = [S_E, p=0]   U2 = [S_E, p=2]   U3 = [S_E, p=1]   V1 = [S_B, p=1]   V2 = [S_B, p=0]   W = [S_T, p=2]
//   Delta^T_l = pref_l W_l,   Delta^E_l = -2 U1_l + (l+1)(l+2) U2_l - 2 U3_{l+1},
//   Delta^B_l = 2 (l+2) V1_l - 2 V2_{l+1}.
// Those six sums are exactly what the scalar transfer kernel computes (a2 + a3: recurrence in registers,
// tau-sum, reduction), so the tensor path is two runs of the three-source kernels of transfer.cu on a
// plan whose l list is the union of {l} and {l + 1}, fed with
//   run A: (S_E, S_T, S_E / x) -> (U1, pref W, U3)      run B: (S_B, S_E, S_B / x) -> (V2, pref U2, V1)
// (the kernel's second slot carries the 1/x^2 weight and the sqrt((l+2)!/(l-2)!) prefactor), issued as one
// batched launch of two members per cosmology, with a small kernel in front that lays the sources out (and forms S / x) and
// a small kernel behind that combines the rows.  10 FP64
// instructions per executed (l, k, tau) term against the 8 a dedicated six-sum kernel would need; tensor
// runs are small (l_max_tensor = 1500 against l_max_scalar = 11000).
#include <algorithm>

#include "los_internal.cuh"

namespace gcamb {

namespace {

// The two runs go out as ONE batched launch (twice the thread blocks: a finer tail than two launches of n_k
// blocks each), so their sources are laid out as a batch of two per kernel slot and cosmology b:
//   slot 0 = [.. S_E(b) | S_B(b) ..],  slot 1 = [.. S_T(b) | S_E(b) ..],  slot 2 = [.. S_E(b) / x | S_B(b) / x ..]
// (1/x: the plan's rounded reciprocal); member 2 b of the launch is run A of cosmology b, member 2 b + 1 its run B.
__global__ void __launch_bounds__(256) tensor_prep_kernel(const double *__restrict__ S_T, const double *__restrict__ S_E,
                                                          const double *__restrict__ S_B, const double *__restrict__ inv_x,
                                                          double *__restrict__ slot0, double *__restrict__ slot1,
                                                          double *__restrict__ slot2, size_t n)
{
    const size_t in = (size_t)blockIdx.y * n, out = 2 * in;   // cosmology blockIdx.y
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double inv = inv_x[i], t = S_T[in + i], e = S_E[in + i], b = S_B[in + i];
        slot0[out + i] = e;       slot0[out + n + i] = b;
        slot1[out + i] = t;       slot1[out + n + i] = e;
        slot2[out + i] = e * inv; slot2[out + n + i] = b * inv;
    }
}

// raw: [B][2 runs][3][n_le][n_k] (rows of the union list); Delta: [B][3][n_l][n_k] (rows of the caller's list)
__global__ void __launch_bounds__(256) tensor_combine_kernel(const double *__restrict__ raw,
                                                             const int32_t *__restrict__ pos0, const int32_t *__restrict__ pos1,
                                                             const double *__restrict__ cE, const double *__restrict__ cB,
                                                             double *__restrict__ Delta, int n_l, int n_le, int n_k)
{
    const int a = blockIdx.y;
    const size_t r0 = (size_t)pos0[a] * n_k, r1 = (size_t)pos1[a] * n_k, plane = (size_t)n_le * n_k;
    const double *rawA = raw + (size_t)blockIdx.z * 6 * plane, *rawB = rawA + 3 * plane;
    const double ce = cE[a], cb = cB[a];
    const size_t oplane = (size_t)n_l * n_k, out = (size_t)blockIdx.z * 3 * oplane + (size_t)a * n_k;
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_k; j += gridDim.x * blockDim.x) {
        const double U1 = rawA[r0 + j], pW = rawA[plane + r0 + j], U3n = rawA[2 * plane + r1 + j];
        const double V2n = rawB[r1 + j], pU2 = rawB[plane + r0 + j], V1 = rawB[2 * plane + r0 + j];
        Delta[out + j] = pW;
        Delta[oplane + out + j] = fma(ce, pU2, -2.0 * U1) - 2.0 * U3n;
        Delta[2 * oplane + out + j] = fma(cb, V1, -2.0 * V2n);
    }
}

}  // namespace

size_t tensor_work_bytes(const gcamb_los_plan *p)
{
    return sizeof(double) * (6 * (size_t)p->n_k * p->n_tau + 6 * (size_t)p->n_l * p->n_k);
}

gcamb_status launch_transfer_tensor(const gcamb_los_plan *p, int n_batch, const double *S_T, const double *S_E,
                                    const double *S_B, double *Delta, double *work, cudaStream_t stream)
{
    const size_t n_pt = (size_t)p->n_k * p->n_tau, B = (size_t)n_batch;
    double *slot0 = work, *slot1 = work + 2 * B * n_pt, *slot2 = work + 4 * B * n_pt, *raw = work + 6 * B * n_pt;
    const unsigned blocks = (unsigned)std::min<size_t>((n_pt + 255) / 256, (size_t)p->n_sm * 16);
    tensor_prep_kernel<<<dim3(blocks, (unsigned)n_batch), 256, 0, stream>>>(S_T, S_E, S_B, p->d_inv, slot0, slot1, slot2, n_pt);
    GCAMB_CUDA(cudaGetLastError());
    // member 2 b = run A of cosmology b, member 2 b + 1 = its run B: raw [B][2][3][n_le][n_k]
    gcamb_status st = launch_transfer(p, 2 * n_batch, slot0, slot1, slot2, raw, stream);
    if (st != GCAMB_OK) return st;
    dim3 grid((unsigned)std::min((p->n_k + 255) / 256, 64), (unsigned)p->n_l_out, (unsigned)n_batch);
    tensor_combine_kernel<<<grid, 256, 0, stream>>>(raw, p->d_t_pos0, p->d_t_pos1, p->d_t_cE, p->d_t_cB,
                                                    Delta, p->n_l_out, p->n_l, p->n_k);
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

}  // namespace gcamb
