// fused.cu -- sources of a BATCH of cosmologies -> C_l, in one kernel that never writes Delta
// (the emulator use-case of PAPER.md:24, 248; Eq. 1-3).
//
// For the cosmologies of a batch x = k (tau0 - tau) is the same (one plan), so
//   * the coefficient and the recurrence step  f_{l-1} = (2l+1)/x f_l - f_{l+1}  are issued ONCE
//     per (l, k, tau) and shared by all cosmologies of a block of BC, and
//   * the tau-sum  Delta^X_l(k; b) = sum_i j_l(x_i) s_X(b; tau_i)  IS a dense contraction
//     [l-tile x tau] . [tau x (X, b)]: it runs on the FP64 tensor cores (mma.sync.m8n8k4.f64, DMMA).
//     On B200 DMMA has the SAME peak as DFMA (measured: both 64 FMA/clk/SM, and mixed streams add
//     up to one pipe's worth: profiles/README.md), so the gain is not a second pipe but (a) one
//     issue slot per 256 FMAs instead of 8 two-cycle DFMA issues with their register-operand
//     stalls, (b) the cross-lane (tau) reduction happens inside the MMA: no transposing warp
//     reduction, and (c) 2 + 2 BC FP64 lane-slots per (l, k, tau) for BC cosmologies instead of 4 BC.
//
// Mapping: one CTA of 8 warps takes a k row and BC = 4 NB cosmologies; thread = T (k, tau) points
// as in transfer.cu (lanes <-> 32 consecutive tau of a warp slot), recurrence state in registers.
// Per l-tile (V = 8) and started slot a thread runs its 8 recurrence steps and writes j_l .. j_{l-7}
// to a per-warp shared-memory tile [8][32 tau]; the warp reads it back as four A-fragment pairs
// (rows = l, columns = 4 tau) and multiplies them with the B fragments it holds in registers for
// the whole walk: the pre-weighted sources s_X(b; tau) of its own 32 tau, columns (b, X).  The D
// fragments (8 l x 8 columns each) accumulate over the slots of the warp; the eight warps' tiles
// meet in the ring of transfer.cu (mbarrier-paced, flushed one group late).
//
// Eq. 1 is folded into the flush: a thread owns one (l, b) of the group, sums the warps in fixed
// order, applies the Delta^E prefactor and adds  w_b(k) Delta^X Delta^Y  to the CTA's own slice of
// partial spectra in global memory (L2-resident, plain load/add/store: the CTA is the only writer).
// A CTA walks a STATIC list of k rows (balanced by cost at plan creation), so the order of every sum
// is fixed: results are bit-reproducible.  A last small kernel adds the slices in bin order and
// multiplies by 4 pi.
#include <algorithm>
#include <atomic>

#include "los_internal.cuh"
#include "mbar.cuh"

namespace gcamb {

namespace {

struct FusedParams {
    const double *S_T, *S_E;   // [B][n_k][n_tau]
    const double *P_R;         // [B][n_k]
    double *Cpart;             // [n_cblk][n_bins][3][n_l][BC]
    const double *k, *chi, *w, *pref, *inv_x, *dlnk;
    const double2 *start;
    const int32_t *tile, *l_index, *bin_start, *bin_items;
    const uint32_t *tile_mask;   // sparse l lists: bit t % 32 of word t / 32 = tile t holds a listed l
    int n_k, n_tau, n_l, l_min, l_max, n_tiles, n_batch, n_bins, l_contig;
};

constexpr unsigned FULL = 0xffffffffu;
constexpr int NEVER = 0x7fffffff;
constexpr int F_V = 8;          // l-tile = rows of an MMA
constexpr int F_W = 8;          // warps per CTA
constexpr int F_THREADS = 32 * F_W;
constexpr int F_G = 4;          // tiles per ring group: G * V * BC (l, b) pairs = one per thread at BC = 8
constexpr int F_RD = 3;         // ring stages
constexpr int F_LAG = 1;
constexpr int F_JS = 40;        // row stride of the j_l tile: 16-byte fragment loads of a quarter-warp hit 32 distinct banks

__device__ __forceinline__ void dmma(double (&d)[2], double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

// The recurrence alone on one l-tile for the first NA slots of a thread (tiles without a listed l of the SPARSE
// kernel): NA chains interleaved (l outer, slot inner), compensated coefficient as in the MMA path.
template <int NA, int T>
__device__ __forceinline__ void fused_walk(double tl0, const double *my_ix, const double *my_ixlo, double (&fa)[T], double (&fb)[T])
{
    static_assert(T <= 10, "the dispatch on the number of started slots is written out for T <= 10");
    double ixr[NA], er[NA];
#pragma unroll
    for (int j = 0; j < NA; ++j) {
        ixr[j] = my_ix[j * F_THREADS];
        er[j] = tl0 * my_ixlo[j * F_THREADS];
    }
#pragma unroll
    for (int s = 0; s < F_V; ++s) {
        const double tl = tl0 - 2.0 * s;
#pragma unroll
        for (int j = 0; j < NA; ++j) {
            const double c = fma(tl, ixr[j], er[j]);
            const double fn = fma(c, fb[j], -fa[j]);
            fa[j] = fb[j];
            fb[j] = fn;
        }
    }
}

template <int NB, int T> constexpr size_t fused_smem_bytes()
{
    constexpr int P = F_V * 8 * NB;
    return sizeof(double2) * T * F_THREADS                       // start pairs
         + sizeof(double) * 2 * T * F_THREADS                    // 1/x and its rounding residual
         + sizeof(double) * F_W * 2 * F_V * F_JS                 // j_l tiles, double-buffered per warp
         + sizeof(double) * (F_RD * F_G * F_W * P + 2 * F_RD)    // ring + its barriers
         + sizeof(int) * (T * F_THREADS + F_W * 2 * T);          // start tiles, slot windows
}

// NB = 8-column blocks of the contraction: BC = 4 NB cosmologies x (T, E).  T = points per thread.
// SPARSE (l lists with l-tiles that hold no listed l: CAMB's default l sampling): such a tile is
// walked by the recurrence alone (16 FP64 instructions per started slot instead of those plus 16 MMAs), nothing of
// it enters the ring, and its rows are skipped by the flush (the groups of tiles keep their places in the ring:
// taking the groups without a listed l out of the barrier protocol measured 16.0 against 13.3 ms, registers).
// A kernel of its own: the dense kernel is unchanged.
template <int NB, int T, bool SPARSE>
__global__ void __launch_bounds__(F_THREADS, 1) fused_kernel(const FusedParams p)
{
    constexpr int V = F_V, W = F_W, G = F_G, RD = F_RD, LAG = F_LAG, JS = F_JS;
    constexpr int BC = 4 * NB;
    constexpr int P = V * 2 * BC;        // ring entries per warp and tile: [row][b][X]
    constexpr int NPAIR = G * V * BC;    // (l, b) pairs per group
    static_assert(NPAIR <= F_THREADS, "one (l, b) pair per thread at the flush");
    extern __shared__ double2 smem2[];
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __reduce_min_sync(FULL, tid >> 5);
    double2 *my_start = smem2 + tid;                                  // [j * THREADS]
    double *base = reinterpret_cast<double *>(smem2 + (size_t)T * F_THREADS);
    double *my_ix = base + tid;                                       // [j * THREADS]
    double *my_ixlo = base + (size_t)T * F_THREADS + tid;
    base += 2 * (size_t)T * F_THREADS;
    double *jt = base + (size_t)warp * 2 * V * JS;                    // [2][V][JS]
    base += (size_t)W * 2 * V * JS;
    double *ring = base;                                              // [RD][G][W][P]
    base += (size_t)RD * G * W * P;
    const uint32_t bar_full = (uint32_t)__cvta_generic_to_shared(base);
    const uint32_t bar_empty = bar_full + 8 * RD;
    int *my_tile = reinterpret_cast<int *>(base + 2 * RD) + tid;      // [j * THREADS]
    int *slot_win = reinterpret_cast<int *>(base + 2 * RD) + (size_t)T * F_THREADS + warp * 2 * T;

    const int bin = blockIdx.x, cb = blockIdx.y, b0 = cb * BC;
    double *cpart = p.Cpart + ((size_t)cb * p.n_bins + bin) * 3 * p.n_l * BC;   // this CTA's partial spectra [3][n_l][BC]
    for (size_t i = tid; i < (size_t)3 * p.n_l * BC; i += F_THREADS) cpart[i] = 0.0;
    if (tid == 0) for (int d = 0; d < 2 * RD; ++d) mbar_init(bar_full + 8 * d, W);
    __syncthreads();

    // flush: this thread's (tile of the group, row, cosmology)
    const bool f_on = tid < NPAIR;
    const int f_gi = tid / (V * BC), f_r = (tid / BC) % V, f_b = tid % BC;
    // fragment coordinates
    const int fr = lane >> 2, fc = lane & 3;
    const int it0 = p.bin_start[bin], it1 = p.bin_start[bin + 1];

  for (int it = it0; it < it1; ++it) {
    if (it > it0) {   // the ring starts afresh; the partial spectra the other threads stored are visible
        __syncthreads();
        if (tid == 0)
            for (int d = 0; d < 2 * RD; ++d) { mbar_inval(bar_full + 8 * d); mbar_init(bar_full + 8 * d, W); }
        __syncthreads();
    }
    const int kidx = __reduce_min_sync(FULL, p.bin_items[it]);
    const double kval = p.k[kidx];
    const size_t row = (size_t)kidx * p.n_tau;
    // Eq. 1 weight of this k for the flush thread's cosmology
    double f_wk = 0.0;
    if (f_on && b0 + f_b < p.n_batch) f_wk = p.dlnk[kidx] * p.P_R[(size_t)(b0 + f_b) * p.n_k + kidx];
    const int t_begin_load = p.tile[row];   // start tile of the largest x

    // ---- prologue: recurrence state of this thread's points, B fragments of this warp's slots
    double fa[T], fb[T], Bf[T][8][NB];
    int tp[T];
#pragma unroll
    for (int j = 0; j < T; ++j) {
        const int sb = j * F_THREADS + ((warp + j) % W) * 32;   // first tau of this warp's slot j
        const int i = sb + lane;
        const bool valid = i < p.n_tau;
        const int ic = valid ? i : p.n_tau - 1;
        const double inv = p.inv_x[row + ic];
        const double x = __dmul_rn(kval, p.chi[ic]);
        const double res = fma(inv, x, -1.0);               // 1/x = inv + inv_lo, inv_lo = -inv (inv x - 1)
        my_ix[j * F_THREADS] = valid ? inv : 0.0;
        my_ixlo[j * F_THREADS] = valid ? -inv * res : 0.0;
        tp[j] = valid ? p.tile[row + ic] : NEVER;
        my_tile[j * F_THREADS] = tp[j];
        my_start[j * F_THREADS] = p.start[row + ic];
        fa[j] = fb[j] = 0.0;
        // B fragment of MMA m: row (tau) = sb + 8 (m >> 1) + 2 fc + (m & 1), column = 8 nb + fr = (b, X)
#pragma unroll
        for (int m = 0; m < 8; ++m) {
            const int i2 = sb + 8 * (m >> 1) + 2 * fc + (m & 1);
            const bool v2 = i2 < p.n_tau;
            const int ic2 = v2 ? i2 : p.n_tau - 1;
            const double w2 = v2 ? p.w[ic2] : 0.0;
            const double inv2 = p.inv_x[row + ic2];
            const double wx[2] = {w2, w2 * (inv2 * inv2)};   // s_T = w S_T, s_E = w S_E / x^2
#pragma unroll
            for (int nb = 0; nb < NB; ++nb) {
                const int col = 8 * nb + fr, bl = col >> 1, X = col & 1;
                const bool vb = b0 + bl < p.n_batch;
                const int bc = vb ? b0 + bl : p.n_batch - 1;
                const double *S = X ? p.S_E : p.S_T;
                const double v = S[((size_t)bc * p.n_k + kidx) * p.n_tau + ic2];
                Bf[j][m][nb] = vb ? wx[X] * v : 0.0;
            }
        }
    }
#pragma unroll
    for (int j = 0; j < T; ++j) {
        const int first = __reduce_min_sync(FULL, tp[j]);
        const int last = __reduce_max_sync(FULL, tp[j] == NEVER ? -1 : tp[j]);
        if (lane == 0) { slot_win[2 * j] = first; slot_win[2 * j + 1] = last; }
    }
    __syncwarp();
    const int t_begin = __reduce_min_sync(FULL, t_begin_load);
    const int n_walk = p.n_tiles - t_begin;
    // The next row's sources and plan tables on their way into the L2 while this row is walked: with one thread
    // block per SM nothing else covers the DRAM round trips of the prologue above.  SPARSE only: 13.3 -> 13.0 ms;
    // the dense kernel, whose rows take twice as long, measured 23.55 -> 23.68 ms with it.
    if (SPARSE && it + 1 < it1) {
        const int kn = p.bin_items[it + 1];
        const size_t rown = (size_t)kn * p.n_tau;
        const int lines = (p.n_tau * 8 + 127) / 128;                 // 128-byte lines of one source row
        for (int i = tid; i < 2 * BC * lines; i += F_THREADS) {
            const int bl = i / (2 * lines), r = i - bl * 2 * lines, X = r / lines, ln = r - X * lines;
            if (b0 + bl < p.n_batch) {
                const double *src = (X ? p.S_E : p.S_T) + ((size_t)(b0 + bl) * p.n_k + kn) * p.n_tau + (size_t)ln * 16;
                asm volatile("prefetch.global.L2 [%0];" ::"l"(src));
            }
        }
        for (int i = tid; i < 4 * lines; i += F_THREADS) {          // 1/x (8 B), start pairs (16 B), start tiles (4 B) per point
            const char *base = i < lines ? reinterpret_cast<const char *>(p.inv_x + rown)
                             : i < 3 * lines ? reinterpret_cast<const char *>(p.start + rown) - (size_t)lines * 128
                                             : reinterpret_cast<const char *>(p.tile + rown) - (size_t)3 * lines * 128;
            if (i < 3 * lines || (size_t)(i - 3 * lines) * 128 < (size_t)p.n_tau * 4)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(base + (size_t)i * 128));
        }
    }

    // flush of group m: warps summed in index order, Delta^E prefactor, Eq. 1 products into the partial spectra
    // has: some tile of the group holds a listed l (always, unless SPARSE).  A group without one leaves nothing in
    // the ring: its flush neither waits for the other warps nor reads, it only hands the stage back
    auto flush_group = [&](int m, bool has) {
        const int stage = m % RD;
        if (SPARSE && !has) {
            if (lane == 0) mbar_arrive(bar_empty + 8 * stage);
            return;
        }
        const int gcount = min(G, n_walk - m * G);
        // this thread's (l, cosmology) and its three partial spectra: the loads (L2 round trips: the
        // source view showed 8 % of the warp time waiting for them behind the ring sums) are issued
        // before the wait on the ring so that they travel under it
        int li = -1;
        if (f_on && f_gi < gcount) {
            const int l = p.l_max - (t_begin + m * G + f_gi) * V - f_r;
            li = l >= p.l_min ? (p.l_contig ? l - p.l_min : p.l_index[l]) : -1;
        }
        const size_t sp = (size_t)p.n_l * BC;
        double *c = cpart + (size_t)(li >= 0 ? li : 0) * BC + f_b;
        double c0 = 0.0, c1 = 0.0, c2 = 0.0, pf = 0.0;
        if (li >= 0) { c0 = c[0]; c1 = c[sp]; c2 = c[2 * sp]; pf = p.pref[li]; }
        mbar_wait(bar_full + 8 * stage, (m / RD) & 1);
        if (li >= 0) {
            const double2 *e = reinterpret_cast<const double2 *>(
                ring + ((size_t)(stage * G + f_gi) * W) * P + (f_r * BC + f_b) * 2);
            double dT = 0.0, dE = 0.0;
#pragma unroll
            for (int wv = 0; wv < W; ++wv) {
                const double2 v = e[(size_t)wv * (P / 2)];
                dT += v.x;
                dE += v.y;
            }
            dE *= pf;
            const double wT = f_wk * dT, wE = f_wk * dE;
            c[0] = fma(wT, dT, c0);
            c[sp] = fma(wE, dE, c1);
            c[2 * sp] = fma(wT, dE, c2);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * stage);
    };

#define GCAMB_UNI(v) __reduce_min_sync(FULL, (v))
    int na = 0;
    int next_slot = GCAMB_UNI(slot_win[0]);
    int inj = 0, inj_from = next_slot;
    int buf = 0;
    unsigned mask_word = 0, any_hist = 0;   // SPARSE; bit i of any_hist: group n - i holds a listed l
    double tl0 = (double)(2 * (p.l_max - t_begin * V) + 1);
    const int n_groups = (n_walk + G - 1) / G;
    int t = t_begin;
    for (int n = 0; n < n_groups + LAG; ++n) {
      if (n < n_groups) {
        if (n >= RD) mbar_wait(bar_empty + 8 * (n % RD), ((n / RD) - 1) & 1);
        const int gcount = min(G, n_walk - n * G);
        for (int g = 0; g < gcount; ++g, ++t, tl0 -= 2.0 * V) {
            while (next_slot <= t) {
                ++na;
                next_slot = na < T ? GCAMB_UNI(slot_win[2 * na]) : NEVER;
            }
            if (inj_from <= t) {
#pragma unroll
                for (int j = 0; j < T; ++j) {
                    if (my_tile[j * F_THREADS] == t) {
                        const double2 st = my_start[j * F_THREADS];
                        fa[j] = st.x;
                        fb[j] = st.y;
                    }
                }
                while (inj < T && GCAMB_UNI(slot_win[2 * inj + 1]) <= t) ++inj;
                inj_from = inj < T ? GCAMB_UNI(slot_win[2 * inj]) : NEVER;
            }
            double2 *rb = reinterpret_cast<double2 *>(ring + ((size_t)((n % RD) * G + g) * W + warp) * P);
            bool listed = true;
            if constexpr (SPARSE) {
                if ((t & 31) == 0 || t == t_begin) mask_word = GCAMB_UNI(p.tile_mask[t >> 5]);
                listed = (mask_word >> (t & 31)) & 1u;
                any_hist |= (unsigned)listed;
            }
            if (SPARSE && !listed) {
                // a2 alone for the started slots: no tile of j_l, no MMA, no ring entry.  One body per number of
                // started slots (a run-time bound inside the unrolled loops turns into selects on every state register)
#define GCAMB_FW(n) case n: if constexpr (T >= n) fused_walk<n, T>(tl0, my_ix, my_ixlo, fa, fb); break;
                switch (na) {
                    GCAMB_FW(1) GCAMB_FW(2) GCAMB_FW(3) GCAMB_FW(4) GCAMB_FW(5)
                    GCAMB_FW(6) GCAMB_FW(7) GCAMB_FW(8) GCAMB_FW(9) GCAMB_FW(10)
                }
#undef GCAMB_FW
            } else if (na > 0) {
                double D[2][NB][2];   // even / odd MMAs accumulate apart: 2 NB independent chains
#pragma unroll
                for (int h = 0; h < 2; ++h)
#pragma unroll
                    for (int nb = 0; nb < NB; ++nb) D[h][nb][0] = D[h][nb][1] = 0.0;
                // a2 for one slot: eight steps of the recurrence; j_l, .., j_{l-7} of this lane's tau go to tile `b`
                auto recur = [&](int j, int b) {   // j is a constant once the slot loop is unrolled
                    const double ixj = my_ix[j * F_THREADS];
                    const double e = tl0 * my_ixlo[j * F_THREADS];
                    double *tile_w = jt + (size_t)b * V * JS + lane;
#pragma unroll
                    for (int s = 0; s < V; ++s) {
                        const double tl = tl0 - 2.0 * s;
                        const double c = fma(tl, ixj, e);        // correctly rounded (2l+1)/x
                        tile_w[s * JS] = fb[j];
                        const double fn = fma(c, fb[j], -fa[j]);
                        fa[j] = fb[j];
                        fb[j] = fn;
                    }
                };
                // Software pipeline over the slots: the recurrence of slot j + 1 (a dependent chain of 16 FP64
                // instructions, latency-bound on its own) is issued between the A-fragment loads and the 16 MMAs
                // of slot j, which do not depend on it; two tiles suffice (the __syncwarp orders the writes of
                // slot j + 1 behind the reads of slot j - 1).
                recur(0, buf);
#pragma unroll
                for (int j = 0; j < T; ++j) {
                    if (j < na) {
                        __syncwarp();
                        // a3: A fragments (row = l-row fr, column = tau 8 mm + 2 fc + {0,1}) x B fragments
                        const double2 *tile_r = reinterpret_cast<const double2 *>(jt + (size_t)buf * V * JS + fr * JS + 2 * fc);
                        double2 a[4];
#pragma unroll
                        for (int mm = 0; mm < 4; ++mm) a[mm] = tile_r[4 * mm];
                        // unconditional (a slot that has not started carries zeros and yields zeros): no branch between
                        // the chain and the MMAs, so that the scheduler may interleave them
                        if (j + 1 < T) recur(j + 1 < T ? j + 1 : 0, buf ^ 1);
#pragma unroll
                        for (int mm = 0; mm < 4; ++mm) {
#pragma unroll
                            for (int nb = 0; nb < NB; ++nb) {
                                dmma(D[0][nb], a[mm].x, Bf[j][2 * mm][nb]);
                                dmma(D[1][nb], a[mm].y, Bf[j][2 * mm + 1][nb]);
                            }
                        }
                        buf ^= 1;
                    }
                }
                // D fragment: row fr, columns 2 fc, 2 fc + 1 of block nb = (T, E) of cosmology 4 nb + fc
#pragma unroll
                for (int nb = 0; nb < NB; ++nb)
                    rb[fr * BC + 4 * nb + fc] = make_double2(D[0][nb][0] + D[1][nb][0], D[0][nb][1] + D[1][nb][1]);
            } else {
                for (int idx = lane; idx < P / 2; idx += 32) rb[idx] = make_double2(0.0, 0.0);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_full + 8 * (n % RD));
      }
      if (n >= LAG) flush_group(n - LAG, (any_hist >> LAG) & 1u);
      any_hist <<= 1;
    }
#undef GCAMB_UNI
  }   // k rows of this bin
}

// C_l[b][XY][l] = 4 pi sum over bins (in bin order) of the partial spectra
__global__ void __launch_bounds__(256) fused_finish_kernel(const double *__restrict__ Cpart, double *__restrict__ Cl,
                                                           int n_bins, int n_l, int n_batch, int BC)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int cb = blockIdx.y;
    const size_t slice = (size_t)3 * n_l * BC;
    if (idx >= slice) return;
    const int bl = (int)(idx % BC);
    const int li = (int)((idx / BC) % n_l);
    const int spec = (int)(idx / ((size_t)BC * n_l));
    const int b = cb * BC + bl;
    if (b >= n_batch) return;
    const double *src = Cpart + (size_t)cb * n_bins * slice + idx;
    double s = 0.0;
    for (int bin = 0; bin < n_bins; ++bin) s += src[(size_t)bin * slice];
    Cl[((size_t)b * 3 + spec) * n_l + li] = 4.0 * 3.14159265358979323846 * s;
}

template <int NB, int T, bool SPARSE>
gcamb_status launch_sp(const FusedParams &prm, int n_cblk, int device, cudaStream_t stream)
{
    constexpr size_t smem = fused_smem_bytes<NB, T>();
    static_assert(smem <= 227 * 1024, "shared memory of the fused kernel");
    static std::atomic<unsigned long long> attr_done;
    const unsigned long long dev_bit = 1ull << (device & 63);
    if (!(attr_done.load(std::memory_order_acquire) & dev_bit)) {
        GCAMB_CUDA(cudaFuncSetAttribute(fused_kernel<NB, T, SPARSE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_done.fetch_or(dev_bit, std::memory_order_release);
    }
    fused_kernel<NB, T, SPARSE><<<dim3((unsigned)prm.n_bins, (unsigned)n_cblk), F_THREADS, smem, stream>>>(prm);
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

template <int NB, int T>
gcamb_status launch_one(const FusedParams &prm, int n_cblk, int device, cudaStream_t stream)
{
    return prm.tile_mask ? launch_sp<NB, T, true>(prm, n_cblk, device, stream) : launch_sp<NB, T, false>(prm, n_cblk, device, stream);
}

}  // namespace

// Largest n_tau the fused kernel holds in registers for a block of 8 (NB = 2) / 4 (NB = 1) cosmologies
constexpr int FUSED_T_MAX_NB2 = 5, FUSED_T_MAX_NB1 = 10;

bool fused_supported(const gcamb_los_plan *p, int n_batch)
{
    return p->n_src == 2 && !p->curved && n_batch >= 2 && p->n_tau <= F_THREADS * FUSED_T_MAX_NB1;
}

int fused_block(const gcamb_los_plan *p, int n_batch)
{
    return (n_batch > 4 && p->n_tau <= F_THREADS * FUSED_T_MAX_NB2) ? 8 : 4;
}

size_t fused_scratch_bytes(const gcamb_los_plan *p, int n_batch)
{
    const int BC = fused_block(p, n_batch), n_cblk = (n_batch + BC - 1) / BC;
    return sizeof(double) * (size_t)n_cblk * p->n_bins * 3 * p->n_l * BC;
}

gcamb_status launch_fused(const gcamb_los_plan *p, int n_batch, const double *S_T, const double *S_E,
                          const double *P_R, double *scratch, double *Cl, cudaStream_t stream)
{
    FusedParams prm;
    prm.S_T = S_T; prm.S_E = S_E; prm.P_R = P_R; prm.Cpart = scratch;
    prm.k = p->d_k; prm.chi = p->d_chi; prm.w = p->d_w; prm.pref = p->d_pref; prm.inv_x = p->d_inv; prm.dlnk = p->d_dlnk;
    prm.start = p->d_start; prm.tile = p->d_tile; prm.l_index = p->d_l_index;
    prm.bin_start = p->d_bin_start; prm.bin_items = p->d_bin_items; prm.tile_mask = p->d_tile_mask;
    prm.n_k = p->n_k; prm.n_tau = p->n_tau; prm.n_l = p->n_l; prm.l_min = p->l_min; prm.l_max = p->l_max;
    prm.n_tiles = p->n_tiles; prm.n_batch = n_batch; prm.n_bins = p->n_bins;
    prm.l_contig = p->n_l == p->l_max - p->l_min + 1;
    const int BC = fused_block(p, n_batch), n_cblk = (n_batch + BC - 1) / BC;
    const int T = (p->n_tau + F_THREADS - 1) / F_THREADS;
    gcamb_status st = GCAMB_EINVAL;
    if (BC == 8) {
        switch (T) {
            case 1: st = launch_one<2, 1>(prm, n_cblk, p->device, stream); break;
            case 2: st = launch_one<2, 2>(prm, n_cblk, p->device, stream); break;
            case 3: st = launch_one<2, 3>(prm, n_cblk, p->device, stream); break;
            case 4: st = launch_one<2, 4>(prm, n_cblk, p->device, stream); break;
            case 5: st = launch_one<2, 5>(prm, n_cblk, p->device, stream); break;
            default: set_error("fused kernel: n_tau %d too large for a block of 8", p->n_tau); return GCAMB_EINVAL;
        }
    } else {
        switch ((T + 1) / 2) {
            case 1: st = launch_one<1, 2>(prm, n_cblk, p->device, stream); break;
            case 2: st = launch_one<1, 4>(prm, n_cblk, p->device, stream); break;
            case 3: st = launch_one<1, 6>(prm, n_cblk, p->device, stream); break;
            case 4: st = launch_one<1, 8>(prm, n_cblk, p->device, stream); break;
            case 5: st = launch_one<1, 10>(prm, n_cblk, p->device, stream); break;
            default: set_error("fused kernel: n_tau %d too large", p->n_tau); return GCAMB_EINVAL;
        }
    }
    if (st != GCAMB_OK) return st;
    const size_t slice = (size_t)3 * p->n_l * BC;
    fused_finish_kernel<<<dim3((unsigned)((slice + 255) / 256), (unsigned)n_cblk), 256, 0, stream>>>(
        scratch, Cl, p->n_bins, p->n_l, n_batch, BC);
    GCAMB_CUDA(cudaGetLastError());
    return GCAMB_OK;
}

}  // namespace gcamb
