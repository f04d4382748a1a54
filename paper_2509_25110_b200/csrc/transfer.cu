// transfer.cu -- steps a1-a3 of the hot path: sources -> Delta^X_l(k)  (Eq. 2-3).
//
// Mapping: one CTA per k, lanes <-> consecutive tau.
// Every thread carries T (k,tau) points ("slots") whose recurrence state lives in registers for
// the whole walk: f_{l+1}, f_l, 1/x and the pre-weighted sources s_X = w S_X (s_E also / x^2).
// The CTA walks l DOWNWARD in tiles of V; per point and l it issues
//     c   = (2l+1) * (1/x)                  1 DMUL
//     acc_X[l] += s_X * f_l                 n_src DFMA
//     f_{l-1} = c * f_l - f_{l+1}           1 DFMA
// i.e. 2 + n_src FP64 issue slots per executed (l,k,tau) term, no j_l table, no sincos: the start
// pair of each point comes from the plan (plan.cu) and is injected when the walk reaches the
// point's first tile; until then the point carries f = 0 and contributes exactly 0 (R16).
//
// Ragged work: x falls with tau, so within a warp slot j starts no earlier than slot j-1.  The
// tile body is instantiated for every number NA of started slots (warp-uniform), so slots that
// have not started cost nothing and started ones always run as NA interleaved chains.
//
// Reduction: after a tile the V x n_src per-thread sums are reduced across the warp through a
// shared-memory transpose (1 DADD per l and source, no shuffles or selects) into a ring;
// every G tiles the warps' entries are summed in fixed order, the Delta^E prefactor is applied and
// the result stored.
//
// tau ranges longer than one CTA's slots (n_tau > threads * T) are taken in PASSES by the same CTA:
// pass 0 stores its sums, pass p > 0 adds its own to what the CTA stored before (plain loads and
// stores of its own k column, ordered by a CTA barrier).  No atomics, no cleared output buffer: the
// order of every sum is fixed by (n_tau, n_src) alone, so results are bit-reproducible run to run,
// a k row does not depend on the other rows, and the batched call equals a loop of single calls.
#include <algorithm>
#include <atomic>
#include <cassert>

#include "los_internal.cuh"
#include "mbar.cuh"

// compute-sanitizer is not available on the target pool: a build with -DGCAMB_DEBUG (GCAMB_DEBUG=1
// python -m paper_2509_25110_b200.build --force) checks every global and ring index of the transfer
// kernel with device asserts instead; the GPU tests are run once against that build per change.
#ifdef GCAMB_DEBUG
#define GCAMB_ASSERT(c) assert(c)
#else
#define GCAMB_ASSERT(c) ((void)0)
#endif

namespace gcamb {

struct TransferParams {
    const double *S[4];   // NSRC = 4 (tensor plans): sums of the kinds of S[0], S[1], S[0], S[1] again
    double *Delta;
    const double *k, *chi, *w, *pref, *inv_x;
    const double2 *start;
    const int32_t *tile, *korder, *l_index, *l_list, *kz;
    const uint32_t *tile_mask;   // [ceil(n_tiles/32)] bit = the tile holds an l of the list (sparse lists only)
    int n_k, n_tau, n_l, l_min, l_max, n_tiles, n_batch, n_pass, pass_len;
    int overlap_prev;   // host side only: the first launch of this range may overlap the launch before it (programmatic stream serialization)
    int order_reversed;   // korder[r] == n_k - 1 - r
    int l_contig;   // l_list = l_min .. l_max without gaps: position of l is l - l_min
    int k_first;    // this launch covers positions k_first .. k_first + gridDim.x/n_batch - 1 of korder
    int zero_fill;  // this launch also zeroes the skipped region of Delta (all rows of it)
    // open-universe plans (CURVED kernels, reading R28); appended so that the flat kernels see the same layout
    const double *cth, *s2, *ib2;   // coth(chi_i), 1/sinh^2(chi_i) [n_tau]; 1/beta_j^2 [n_k]
    const double2 *coef;            // [n_k][n_tiles V] (A_l, R_l) of the step Phi_{l-1} = A_l coth(chi) Phi_l - R_l Phi_{l+1}
    const int32_t *l_end;           // [n_k] closed universes: Delta_l(k) = 0 for l > l_end[k] = beta_k - 1 (open: INT_MAX)
};

constexpr int T_MAX = 12;      // points per thread: the NA dispatch of the kernel is written out up to 12
constexpr unsigned FULL = 0xffffffffu;
constexpr int NEVER = 0x7fffffff;

// Cross-lane reduction of one tile: every lane holds P = NSRC*V partial sums (acc flattened as
// [q][s]); lane c < P returns the sum over the 32 lanes of partial c, in a fixed order.
// Transposed through a per-warp shared-memory scratch [32][P+2] (the +2 keeps the 16-byte stores
// of a quarter-warp on distinct banks).  With C = the power of two >= P, the warp splits into
// 32/C lane groups; group g sums rows g*C .. g*C+C-1 of column lane%C in four interleaved chains
// (DADD latency, not throughput, bounds a single chain), then the groups are combined by xor
// shuffles: P/2 STS.128 + C LDS.64 + (C + log2(32/C)) DADD per lane, against ~9 issue slots per
// partial for a shuffle butterfly -- on sm_100a an FP64 instruction holds its sub-partition's
// issue port for two cycles and nothing co-issues with it, so every other instruction costs
// FP64 time (profiles/README.md, "machine model").
template <int P>
__device__ __forceinline__ double warp_transpose_reduce(const double *vals, double *scratch, int lane)
{
    constexpr int RS = P + 2;
    constexpr int C = P <= 8 ? 8 : (P <= 16 ? 16 : 32);   // columns per lane group
    constexpr int ROWS = C;                               // rows per lane group = 32 / (32 / C)
    static_assert(P <= 32 && P % 2 == 0, "one column per lane");
    double2 *row = reinterpret_cast<double2 *>(scratch + lane * RS);
#pragma unroll
    for (int i = 0; i < P / 2; ++i) row[i] = make_double2(vals[2 * i], vals[2 * i + 1]);
    __syncwarp();
    const int col = lane & (C - 1), grp = lane / C;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    if (col < P) {
        const double *base = scratch + (size_t)grp * ROWS * RS + col;
        s0 = base[0];          // not 0.0 + base[0]: the compiler keeps that add (it turns -0 into +0)
        s1 = base[RS];
        s2 = base[2 * RS];
        s3 = base[3 * RS];
#pragma unroll
        for (int r = 4; r < ROWS; r += 4) {
            s0 += base[r * RS];
            s1 += base[(r + 1) * RS];
            s2 += base[(r + 2) * RS];
            s3 += base[(r + 3) * RS];
        }
    }
    double sum = (s0 + s1) + (s2 + s3);
#pragma unroll
    for (int o = C; o < 32; o <<= 1) sum += __shfl_xor_sync(FULL, sum, o);
    __syncwarp();
    return sum;
}

// ---- ring of partial sums between the warps of a CTA, and its shared-memory mbarriers.
// The walk is cut into groups of G tiles; group n lives in ring stage n % RD.  A warp that has
// written its partial sums of group n arrives on full[stage] and then flushes its share of group
// n - LAG, whose full[] barrier has normally completed long before; having read it, it arrives on
// empty[stage], which a warp awaits before it writes group n + RD - LAG ... into that stage again.
// So a warp only ever waits when it is more than a group ahead of the slowest warp of its CTA,
// instead of at every group as with __syncthreads (10 % of the warp time was barrier wait: the
// warps sit on different sub-partitions and have different numbers of started slots).
// Measured: RD = 3, LAG = 1 best (-2 %); more stages or more lag are slower.
constexpr int RD = 3;    // ring stages
constexpr int LAG = 1;   // a group is flushed this many groups after it was written (<= RD - 2)

// a2 + a3 for one l-tile and the first NA slots of this thread: NA independent recurrence chains.
// Slots are taken one after the other (j outer, l inner): the V recurrence steps of a slot form
// one dependent chain (DMUL + DFMA per step on the plain rows, 8 cycles each, measured), which the
// other slots' instructions and the other resident warps cover; ptxas interleaves the slots (l
// outer) whatever the source order, which is what lets consecutive instructions share operands.
//
// COMP (reading R14): c = (2l+1) * fl(1/x) carries the relative
// error r of the rounded reciprocal into EVERY step with the same sign, i.e. the walk follows
// j_l(x (1 - r)): a phase error x r of up to x 2^-53 that the tau-sum's cancellation multiplies.
// The compensated body adds the reciprocal's rounding residual: c = fma(2l+1, inv, e) with
// e = (2l_top+1) * inv_lo taken once per tile (inv_lo ~ 1e-16 inv: its change inside a tile is
// far below an ulp of c), which makes c the correctly rounded quotient.
// CURVED (open universe, reading R28): the step is Phi_{l-1} = A_l coth(chi) Phi_l - R_l Phi_{l+1} with the
// per-(k, l) coefficients cf[s] = (A_l, R_l) of the plan and ix = coth(chi): one DMUL more per term.
template <int NA, int T, int V, int NSRC, bool COMP, bool CURVED, bool QFORM>
__device__ __forceinline__ void tile_body(double tl0, const double2 (&cf)[V], const double (&ix)[T], const double *ixlo, int stride,
                                          const double (&src)[NSRC][T], double (&fa)[T], double (&fb)[T],
                                          double (&acc)[NSRC][V])
{
#pragma unroll
    for (int j = 0; j < NA; ++j) {
        double e = 0.0;
        if (COMP) e = tl0 * ixlo[j * stride];
#pragma unroll
        for (int s = 0; s < V; ++s) {
            const double tl = CURVED ? cf[s].x : tl0 - 2.0 * s;   // 2l+1  (curved: (2l+1)/b_l)
            // QFORM (plain single-pass rows): the product is taken as (2l+1) * (f_l / x), not as
            // ((2l+1) / x) * f_l.  The operand the slots share, 2l+1, then sits in the three-operand DFMA,
            // where the operand cache (.reuse) saves a register fetch, instead of in the two-operand DMUL,
            // which is at its two cycles anyway (an FP64 instruction costs max(2, register operands
            // fetched) cycles: profiles/README.md 6.7).  Measured: config 1 -1.3 %, config 2 -0.6 %, sparse
            // l lists -2.1 %, open universe -1.6 %; the multi-pass kernels of config 4 +0.4 %: they and the
            // compensated rows keep the coefficient form.
            const double c = COMP ? fma(tl, ix[j], e) : (QFORM ? ix[j] * fb[j] : tl * ix[j]);
#pragma unroll
            for (int q = 0; q < NSRC; ++q) acc[q][s] = fma(src[q][j], fb[j], acc[q][s]);
            const double fa_w = CURVED ? cf[s].y * fa[j] : fa[j];
            const double fn = QFORM ? fma(tl, c, -fa_w) : fma(c, fb[j], -fa_w);
            fa[j] = fb[j];
            fb[j] = fn;
        }
    }
}

// A tile none of whose l is in the l list (sparse lists, R21: CAMB's default l sampling computes
// about every 50th l): only the recurrence walks it, 2 FP64 instructions per term, no accumulators,
// no reduction.  The NA chains are interleaved (l outer, slot inner): without the accumulates a
// single slot's 8-step DFMA chain would be latency-bound.
template <int NA, int T, int V, bool COMP, bool QFORM>
__device__ __forceinline__ void tile_body_walk(double tl0, const double (&ix)[T], const double *ixlo, int stride,
                                               double (&fa)[T], double (&fb)[T])
{
    double e[NA];
    if (COMP) {
#pragma unroll
        for (int j = 0; j < NA; ++j) e[j] = tl0 * ixlo[j * stride];
    }
#pragma unroll
    for (int s = 0; s < V; ++s) {
        const double tl = tl0 - 2.0 * s;
#pragma unroll
        for (int j = 0; j < NA; ++j) {
            const double c = COMP ? fma(tl, ix[j], e[j]) : (QFORM ? ix[j] * fb[j] : tl * ix[j]);
            const double fn = QFORM ? fma(tl, c, -fa[j]) : fma(c, fb[j], -fa[j]);
            fa[j] = fb[j];
            fb[j] = fn;
        }
    }
}

// MULTI: the tau range takes several passes (n_tau > threads * T).  A kernel of its own, so that the
// single-pass kernels carry neither the pass loop nor the load-add-store of the flush (measured:
// config 1 +4 % with a run-time pass count).
template <int T, int V, int NSRC, int G, int MAXTHREADS, int MINBLOCKS, bool COMP, bool SPARSE, bool MULTI, bool CURVED>
__global__ void __launch_bounds__(MAXTHREADS, MINBLOCKS) transfer_kernel(const TransferParams p)
{
    static_assert(!(CURVED && (COMP || SPARSE)), "the open-universe kernels are dense and uncompensated");
    static_assert(T >= 1 && T <= T_MAX, "the NA dispatch below is written out for T <= 12");
    constexpr int P = NSRC * V;          // partial sums per thread and tile
    constexpr int NOUT = (G * P + MAXTHREADS - 1) / MAXTHREADS;   // flush outputs per thread (full CTA)
    // Shared memory, laid out with the compile-time strides of a full CTA (NT threads, WM warps) whatever
    // blockDim is, so that every address is a constant offset from a per-thread base:
    // start pairs [T][NT] | transpose scratch [WM][32][P+2] | ring [RD][G][WM][P] | barriers [2 RD] |
    // start tiles [T][NT] | slot first/last start tile [WM][2T] | (COMP) reciprocal residuals [T][NT]
    constexpr int NT = MAXTHREADS, WM = NT / 32;
    extern __shared__ double2 smem2[];
    const int tid = threadIdx.x, lane = tid & 31, W = blockDim.x >> 5;
    const int warp = __reduce_min_sync(0xffffffffu, tid >> 5);   // through a warp reduction: uniform register
    double2 *my_start = smem2 + tid;     // [j * NT]: private to this thread, no barrier needed
    double *scratch = reinterpret_cast<double *>(smem2 + (size_t)T * NT) + (size_t)warp * 32 * (P + 2);
    double *ring = reinterpret_cast<double *>(smem2 + (size_t)T * NT) + (size_t)WM * 32 * (P + 2);
    int *my_tile = reinterpret_cast<int *>(ring + (size_t)RD * G * WM * P + 2 * RD) + tid;   // [j * NT]
    int *slot_win = reinterpret_cast<int *>(ring + (size_t)RD * G * WM * P + 2 * RD) + (size_t)T * NT + warp * 2 * T;
    // compensated rows only: residuals of the rounded reciprocals [T][NT], after the (8-byte aligned) int tables
    double *my_ixlo = reinterpret_cast<double *>(reinterpret_cast<int *>(ring + (size_t)RD * G * WM * P + 2 * RD) +
                                                 (((size_t)T * NT + WM * 2 * T + 1) & ~(size_t)1)) + tid;
    const uint32_t bar_full = (uint32_t)__cvta_generic_to_shared(ring + (size_t)RD * G * WM * P);
    const uint32_t bar_empty = bar_full + 8 * RD;
    // open / closed universes only: this warp's copy of the coefficient pairs of two ring groups [2][G V]
    // (double-buffered: the pairs of group n + 1 are fetched with cp.async while group n is walked; read
    // straight from global memory every tile they cost an L2 round trip per tile: long_scoreboard 1.2 per issue)
    double2 *cfs = reinterpret_cast<double2 *>(reinterpret_cast<int *>(ring + (size_t)RD * G * WM * P + 2 * RD) +
                                               (((size_t)T * NT + WM * 2 * T + 3) & ~(size_t)3)) + (size_t)warp * 2 * G * V;
    if (tid == 0) for (int d = 0; d < 2 * RD; ++d) mbar_init(bar_full + 8 * d, W);
    __syncthreads();
    const int bid = blockIdx.x;
    // The compensated rows run as their own small launch; the launch after it carries the
    // programmatic-stream-serialization attribute and may start as soon as every CTA of this one has
    // passed this point (the two launches write disjoint rows of Delta and never wait on each other;
    // the dependent launch waits for this one at its very end, see griddepcontrol.wait below).
    asm volatile("griddepcontrol.launch_dependents;");
    const int krel = bid / p.n_batch, b = bid - krel * p.n_batch;
    const int krank = p.k_first + krel;   // position in the cost order
    constexpr bool comp = COMP;           // this launch takes the compensated coefficient
    // the cost order is the k grid reversed whenever cost grows with k: no table look-up then
    const int kidx = p.order_reversed ? p.n_k - 1 - krank : __reduce_min_sync(0xffffffffu, p.korder[krank]);   // uniform register, like the bookkeeping below
    const double kval = p.k[kidx];
    const int l_end = CURVED ? p.l_end[kidx] : 0x7fffffff;
    const size_t row = (size_t)kidx * p.n_tau;
    const size_t delta_b = (size_t)b * NSRC * p.n_l;
#define DIDX(q, li) (delta_b + (size_t)(q) * p.n_l + (li)) * p.n_k + kidx

  const int n_pass = MULTI ? p.n_pass : 1;
  for (int pass = 0; pass < n_pass; ++pass) {
    if (MULTI && pass) {   // the ring and its barriers start afresh; the stores of the previous pass are visible to the whole CTA
        __syncthreads();
        if (tid == 0)
            for (int d = 0; d < 2 * RD; ++d) { mbar_inval(bar_full + 8 * d); mbar_init(bar_full + 8 * d, W); }
        __syncthreads();
    }
    const int i_begin = pass * p.pass_len;
    const int i_end = min(p.n_tau, i_begin + p.pass_len);

    // ---- a1: source staging.  Slot j of the CTA covers tau indices i_begin + j*blockDim ...
    // + blockDim - 1 in W chunks of 32 consecutive tau ("ranks"; rank 0 has the largest x and the
    // most work: on the log-spaced part of the tau grid x halves across one slot).  The warps walk
    // the tiles together, so the rank -> warp map rotates with the slot (not with the row: a row's
    // result must not depend on where it sits in the launch) to give
    // every warp the same mix of heavy and light ranks; the lanes of a warp slot are 32 consecutive
    // tau and start within a tile or two of each other (lockstep waste ~1%).
    // zero-prefix lengths of the (at most two, normally) Delta rows this CTA zero-fills: looked up here
    // so that the look-ups travel with the prologue loads instead of adding their own round trips
    const int zf_rows = NSRC * p.n_l, zf_step = gridDim.x / p.n_batch;
    const bool zf = (!MULTI || pass == 0) && p.zero_fill;
    int zf_nz[2] = {0, 0};
#pragma unroll
    for (int u = 0; u < 2; ++u) {
        const int r = krel + u * zf_step;
        if (zf && r < zf_rows) {
            const int li = r % p.n_l;
            zf_nz[u] = p.kz[(p.l_max - (p.l_contig ? p.l_min + li : p.l_list[li])) / V];
        }
    }
    // first tile of this CTA = start tile of its largest x (loaded here, with the rest of the prologue)
    const int t_begin_load = p.tile[row + i_begin];
    double fa[T], fb[T], ix[T], src[NSRC][T];
    // Branch-free: slots past the end of the tau range read a clamped (valid) index and are masked
    // afterwards, so that the ~6 T loads of a thread are all in flight together instead of one
    // slot's round trip to L2/HBM after the other (the prologue was 11 % of the warp time).
    int tp[T];
#pragma unroll
    for (int j = 0; j < T; ++j) {
        const int i = i_begin + j * (int)blockDim.x + ((warp + j) % W) * 32 + lane;
        const bool valid = i < i_end;
        const int ic = valid ? i : i_end - 1;
        const size_t sx = ((size_t)b * p.n_k + kidx) * p.n_tau + ic;
        GCAMB_ASSERT(kidx >= 0 && kidx < p.n_k && b < p.n_batch && ic >= 0 && ic < p.n_tau && krank < p.n_k);
        // 1/x from the plan: no division in the per-call path (open universe: coth(chi), a table over tau)
        const double inv = CURVED ? p.cth[ic] : p.inv_x[row + ic];
        const double w = valid ? p.w[ic] : 0.0;
        fa[j] = fb[j] = 0.0;
        ix[j] = valid ? inv : 0.0;
        if (comp) {   // 1/x = inv + inv_lo,  inv_lo = -inv * (inv x - 1), the residual taken exactly by the fma
            const double x = __dmul_rn(kval, p.chi[ic]);
            const double res = fma(inv, x, -1.0);
            my_ixlo[j * NT] = valid ? -inv * res : 0.0;
        }
        tp[j] = valid ? p.tile[row + ic] : NEVER;
        my_start[j * NT] = p.start[row + ic];   // never injected when the slot is masked (tile NEVER)
        src[0][j] = w * p.S[0][sx];
        src[1][j] = w * p.S[1][sx] * (CURVED ? p.ib2[kidx] * p.s2[ic] : inv * inv);   // 1/x^2 (1/(beta sinh chi)^2)
        if (NSRC >= 3) src[2][j] = w * p.S[2][sx];
        if (NSRC == 4) src[NSRC - 1][j] = w * p.S[3][sx] * (inv * inv);   // tensor plans: a second 1/x^2 sum with the prefactor
        my_tile[j * NT] = tp[j];
    }
#pragma unroll
    for (int j = 0; j < T; ++j) {
        // x falls with tau: within a warp every point of slot j starts no later than any point of
        // slot j+1, so the start windows [first, last] of the slots are ordered
        const int first = __reduce_min_sync(FULL, tp[j]);
        const int last = __reduce_max_sync(FULL, tp[j] == NEVER ? -1 : tp[j]);
        if (lane == 0) { slot_win[2 * j] = first; slot_win[2 * j + 1] = last; }
    }
    __syncwarp();

    const int t_begin = __reduce_min_sync(FULL, t_begin_load);

    // l above the first tile of a k: Delta is exactly zero there (R16).  Those elements form, for
    // every l, a prefix k < kz[tile of l] of the Delta row (x grows with k, so the first tile of a k
    // never rises with k: checked at plan creation), so the CTAs share the rows among themselves and
    // zero them with coalesced stores (a CTA's own zero elements lie along l, 8 bytes every n_k
    // doubles).  Later passes (smaller x) start at or below the first tile of pass 0.
    if (zf) {
        int u = 0;
        for (int r = krel; r < zf_rows; r += zf_step, ++u) {
            const int li = r % p.n_l;
            const int nz = u < 2 ? zf_nz[u < 1 ? 0 : 1]
                                 : p.kz[(p.l_max - (p.l_contig ? p.l_min + li : p.l_list[li])) / V];
            double *dst = p.Delta + (delta_b + r) * p.n_k;
            GCAMB_ASSERT(nz >= 0 && nz <= p.n_k && r < zf_rows && li < p.n_l);
            for (int j = tid; j < nz; j += blockDim.x) dst[j] = 0.0;
        }
    }

    // flush bookkeeping: output `o` of this thread in a G-tile group is ring column
    // idx = tid + o*blockDim -> (tile gi, source q, row s); its l-index and Delta^E prefactor are
    // looked up at the flush (fetching them a group ahead costs registers across the tile loop and
    // measured 0.8 % slower)
    int f_li[NOUT];
    double f_pref[NOUT];
    auto flush_columns = [&](int t_first) {
#pragma unroll
        for (int o = 0; o < NOUT; ++o) {
            const int idx = tid + o * (int)blockDim.x;
            const int gi = idx / P, r = idx - gi * P, q = r / V, s = r - q * V;
            const int l = p.l_max - (t_first + gi) * V - s;
            int li = -1;
            if (idx < G * P && l >= p.l_min) li = p.l_contig ? l - p.l_min : p.l_index[l];
            f_li[o] = li;
            f_pref[o] = ((q == 1 || (NSRC == 4 && q == 3)) && li >= 0) ? p.pref[li] : 1.0;
            if (CURVED && l > l_end) f_pref[o] = 0.0;   // closed universe: no function above beta - 1 (the walk carries a constant there)
        }
    };

    const int n_walk = p.n_tiles - t_begin;
    // flush of group m: the warps' entries summed in fixed order (by warp index), Delta^E prefactor,
    // store.  `has`: some tile of the group holds a listed l (always, unless SPARSE).
    auto flush_group = [&](int m, bool has) {
        const int stage = m % RD;
        const int t_first = t_begin + m * G;
        const int gcount = min(G, n_walk - m * G);
        if (has) {
            flush_columns(t_first);
            mbar_wait(bar_full + 8 * stage, (m / RD) & 1);
            const double *fbuf = ring + (size_t)stage * G * WM * P;
#pragma unroll
            for (int o = 0; o < NOUT; ++o) {
                const int idx = tid + o * (int)blockDim.x;
                const int li = f_li[o];
                if (idx < gcount * P && li >= 0) {
                    const int gi = idx / P, r = idx - gi * P, q = r / V;
                    double sum = 0.0;
                    for (int wv = 0; wv < W; ++wv) sum += fbuf[((size_t)gi * WM + wv) * P + r];
                    sum *= f_pref[o];
                    double *dst = p.Delta + DIDX(q, li);
                    *dst = (MULTI && pass) ? *dst + sum : sum;   // pass p adds to what this CTA stored in passes < p
                }
            }
            // CTAs smaller than the one NOUT was sized for: the remaining columns
            for (int idx = tid + NOUT * (int)blockDim.x; idx < gcount * P; idx += blockDim.x) {
                const int gi = idx / P, r = idx - gi * P, q = r / V, s = r - q * V;
                const int l = p.l_max - (t_first + gi) * V - s;
                const int li = l >= p.l_min ? (p.l_contig ? l - p.l_min : p.l_index[l]) : -1;
                if (li >= 0) {
                    double sum = 0.0;
                    for (int wv = 0; wv < W; ++wv) sum += fbuf[((size_t)gi * WM + wv) * P + r];
                    if (q == 1 || (NSRC == 4 && q == 3)) sum *= p.pref[li];
                    if (CURVED && l > l_end) sum = 0.0;
                    double *dst = p.Delta + DIDX(q, li);
                    *dst = (MULTI && pass) ? *dst + sum : sum;
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * stage);
    };

    int na = 0;                               // started slots of this warp (warp-uniform)
    // warp-uniform bookkeeping is read through warp reductions (CREDUX), which puts it in uniform
    // registers: branches on it need no convergence barrier and it takes no vector registers
#define GCAMB_UNI(v) __reduce_min_sync(FULL, (v))
    int next_slot = GCAMB_UNI(slot_win[0]);   // tile at which slot `na` starts
    int inj = 0;                              // first slot with points still to start (warp-uniform)
    int inj_from = next_slot;                 // its first start tile
    unsigned any_hist = 0;                    // bit i: group n - i holds a listed l (SPARSE; else every group)
    unsigned mask_word = 0;                   // SPARSE: bit (t & 31) of tile_mask[t >> 5] = tile t holds a listed l
    double tl0 = (double)(2 * (p.l_max - t_begin * V) + 1);   // 2l+1 at the top of the tile
    const int n_groups = (n_walk + G - 1) / G;
    int t = t_begin;
    // group n is walked in iteration n and flushed in iteration n + LAG (one call site for the flush)
    for (int n = 0; n < n_groups + LAG; ++n) {
      bool g_any = false;                     // some tile of this group holds a listed l
      if (n < n_groups) {
        g_any = !SPARSE;
        if (n >= RD) mbar_wait(bar_empty + 8 * (n % RD), ((n / RD) - 1) & 1);
        const int gcount = min(G, n_walk - n * G);
        if constexpr (CURVED) {
            auto fetch_group = [&](int m) {   // coefficient pairs of group m -> buffer m & 1 (16 bytes per cp.async)
                const int cnt = min(G, n_walk - m * G) * V;
                const double2 *src = p.coef + ((size_t)kidx * p.n_tiles + t_begin + (size_t)m * G) * V;
                for (int i = lane; i < cnt; i += 32) {
                    const uint32_t dst = (uint32_t)__cvta_generic_to_shared(cfs + (m & 1) * G * V + i);
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src + i) : "memory");
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
            };
            if (n == 0) fetch_group(0);
            if (n + 1 < n_groups) {
                fetch_group(n + 1);
                asm volatile("cp.async.wait_group 1;" ::: "memory");   // group n has landed, n + 1 may be in flight
            } else {
                asm volatile("cp.async.wait_group 0;" ::: "memory");
            }
            __syncwarp();
        }
        for (int g = 0; g < gcount; ++g, ++t, tl0 -= 2.0 * V) {
        while (next_slot <= t) {
            ++na;
            next_slot = na < T ? GCAMB_UNI(slot_win[2 * na]) : NEVER;
        }
        // inject the plan's start pair (j_{lhi+1}, j_lhi) into points whose walk begins here;
        // skipped (warp-uniformly) on the tiles where no slot of this warp is inside its window
        if (inj_from <= t) {
#pragma unroll
            for (int j = 0; j < T; ++j) {
                if (my_tile[j * NT] == t) {
                    const double2 st = my_start[j * NT];
                    fa[j] = st.x;
                    fb[j] = st.y;
                }
            }
            while (inj < T && GCAMB_UNI(slot_win[2 * inj + 1]) <= t) ++inj;
            inj_from = inj < T ? GCAMB_UNI(slot_win[2 * inj]) : NEVER;
        }

        bool acc_on = true;   // this tile holds an l of the list (always, unless SPARSE)
        if constexpr (SPARSE) {
            if ((t & 31) == 0 || t == t_begin) mask_word = __reduce_min_sync(FULL, p.tile_mask[t >> 5]);
            acc_on = (mask_word >> (t & 31)) & 1u;
            g_any |= acc_on;
        }
        double *rb = ring + ((size_t)((n % RD) * G + g) * WM + warp) * P;   // summed by warp index: a fixed order
        GCAMB_ASSERT(g >= 0 && g < G && warp < W && t >= 0 && na <= T && n * G + g == t - t_begin);
        if (SPARSE && !acc_on) {
#define GCAMB_NA(n, C) case n: if constexpr (T >= n) tile_body_walk<n, T, V, C, !C && !MULTI>(tl0, ix, my_ixlo, NT, fa, fb); break;
            switch (na) {
                GCAMB_NA(1, COMP) GCAMB_NA(2, COMP) GCAMB_NA(3, COMP) GCAMB_NA(4, COMP) GCAMB_NA(5, COMP) GCAMB_NA(6, COMP)
                GCAMB_NA(7, COMP) GCAMB_NA(8, COMP) GCAMB_NA(9, COMP) GCAMB_NA(10, COMP) GCAMB_NA(11, COMP) GCAMB_NA(12, COMP)
            }
#undef GCAMB_NA
        } else if (na > 0) {
            double acc[NSRC][V];
#pragma unroll
            for (int q = 0; q < NSRC; ++q)
#pragma unroll
                for (int s = 0; s < V; ++s) acc[q][s] = 0.0;
            double2 cf[V];   // open universe: the tile's V coefficient pairs (the same for every thread of the CTA)
            if constexpr (CURVED) {
                const double2 *cp = cfs + (n & 1) * G * V + g * V;
#pragma unroll
                for (int s = 0; s < V; ++s) cf[s] = cp[s];
            }
#define GCAMB_NA(n, C) case n: if constexpr (T >= n) tile_body<n, T, V, NSRC, C, CURVED, !C && !MULTI>(tl0, cf, ix, my_ixlo, NT, src, fa, fb, acc); break;
#define GCAMB_BODIES(C) switch (na) { \
                GCAMB_NA(1, C) GCAMB_NA(2, C) GCAMB_NA(3, C) GCAMB_NA(4, C) GCAMB_NA(5, C) \
                GCAMB_NA(6, C) GCAMB_NA(7, C) GCAMB_NA(8, C) GCAMB_NA(9, C) GCAMB_NA(10, C) \
                GCAMB_NA(11, C) GCAMB_NA(12, C) }
            GCAMB_BODIES(COMP)
#undef GCAMB_BODIES
#undef GCAMB_NA
            // cross-lane reduction into this warp's ring entry
            const double tot = warp_transpose_reduce<P>(&acc[0][0], scratch, lane);
            if (lane < P) rb[lane] = tot;
        } else {
            for (int idx = lane; idx < P; idx += 32) rb[idx] = 0.0;
        }

        }   // tiles of the group
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_full + 8 * (n % RD));
      }
      any_hist = (any_hist << 1) | (unsigned)g_any;
      if (n >= LAG) flush_group(n - LAG, (any_hist >> LAG) & 1u);
    }
  }   // passes
#undef GCAMB_UNI
#undef DIDX
    // A launch that was started early (programmatic stream serialization) must not COMPLETE before the
    // launch it follows has completed and flushed its stores: later work in the stream orders itself
    // against this launch only.  One CTA suffices to hold the grid open, and it is the last one of the
    // cost order (the lightest row, scheduled last): if every CTA waited here, the early CTAs of the
    // plain launch would sit on their SMs until the compensated launch has finished and nothing would
    // overlap (measured: config 1 0.76 -> 0.88 ms).  No-op for a launch without the attribute.
    if (blockIdx.x == gridDim.x - 1) asm volatile("griddepcontrol.wait;" ::: "memory");
}

// ------------------------------------------------------------------------------------------
constexpr int RING_G = 8;      // tiles between flushes of the ring (4 / 12 / 16 / 24 measured slower)
constexpr int TILE_V = 8;      // l-tile (V = 16 with two resident CTAs measured 3.5 % slower)
constexpr int MINB_128 = 3;    // resident CTAs per SM the <= 128-thread kernels are compiled for (168 registers)
constexpr int MINB_256 = 1;

// Launch shape.  CTA sizes are powers of two of warps (1, 2, 4, 8): the hardware deals
// a CTA's warps round-robin to the SM's four sub-partitions, each with its own FP64 pipe, and a CTA
// advances at the pace of its slowest warp, so warp counts such as 5 leave one pipe with twice the
// work of the others (measured: profiles/README.md).
//   * n_tau <= 128 T_MAX: one pass; least padding wins, at equal padding the smaller CTA, i.e. more
//     points per thread (the cross-thread reduction costs one DADD per thread, tile row and source
//     whatever T is).  Small launches (n_rows CTAs of that shape would leave the SMs' sub-partitions
//     with fewer than FILL_WARPS warps each) trade points per thread for threads until they do: a
//     lone warp per sub-partition runs at the latency of its dependent DFMA chains, not at throughput
//     (config 0: 37 us with one-warp CTAs, 25 us with 128 threads x 3 points).
//   * n_tau <= 256 T_MAX: one pass of a 256-thread CTA (config 2: 14.8 ms against 15.6 ms for two
//     passes of 128 threads).
//   * longer grids: passes of 128 threads x T_MAX points, the last one shorter (config 4: three
//     passes 52.9 ms, two passes of 256 threads 53.4 ms).
// The result depends on (n_tau, n_rows, n_sm) only; the order of every sum depends on the shape, so a
// batched call and a single call agree bit for bit only when they choose the same shape:
// choose_shape is therefore evaluated with the rows of ONE cosmology (n_k), never with n_k * n_batch.
#if !defined(GCAMB_TU_SPARSE) || (GCAMB_TU_SPARSE == 0 && GCAMB_TU_NSRC == 2 && !defined(GCAMB_TU_CURVED))
TransferShape choose_shape(int n_tau, int n_src, long long n_rows, int n_sm)
{
    (void)n_src;
    constexpr int FILL_WARPS = 3;   // per sub-partition (config 1 runs at 3: 3 CTAs x 4 warps per SM)
    auto shape_for = [&](int threads) {
        TransferShape s;
        s.V = TILE_V;
        s.threads = threads;
        s.n_pass = (n_tau + threads * T_MAX - 1) / (threads * T_MAX);
        s.pass_len = s.n_pass > 1 ? threads * T_MAX : n_tau;
        s.T = s.n_pass > 1 ? T_MAX : (n_tau + threads - 1) / threads;
        return s;
    };
    auto padding = [&](const TransferShape &s) { return (long long)s.T * s.threads - n_tau; };
    if (n_tau > 256 * T_MAX) return shape_for(128);
    if (n_tau > 128 * T_MAX) return shape_for(256);
    TransferShape best = shape_for(128);
    for (int threads = 64; threads >= 32; threads >>= 1) {
        const TransferShape s = shape_for(threads);
        if (s.n_pass == 1 && padding(s) <= padding(best)) best = s;
    }
    const long long want = (long long)FILL_WARPS * 4 * n_sm;
    while (best.threads < 256 && best.T >= 4 && n_rows * (best.threads / 32) < want) best = shape_for(best.threads * 2);
    return best;
}
#endif

// One launch over positions [k_first, k_first + n_pos) of the cost order.
template <int T, int V, int NSRC, bool COMP, bool SPARSE, bool CURVED>
static gcamb_status launch_impl(TransferParams prm, const TransferShape &sh, int k_first, int n_pos,
                                bool zero_fill, bool overlap_previous, int device, cudaStream_t stream)
{
    if (n_pos <= 0) return GCAMB_OK;
    prm.k_first = k_first;
    prm.zero_fill = zero_fill;
    // shared memory of a full CTA (the layout uses the compile-time strides whatever the launch size)
    auto smem_bytes = [](int threads) {
        const int W = threads / 32;
        size_t smem = sizeof(double2) * T * threads + sizeof(double) * W * 32 * (NSRC * V + 2) +
                      sizeof(double) * (RD * RING_G * W * NSRC * V + 2 * RD) +
                      sizeof(int) * (((size_t)T * threads + W * 2 * T + 1) & ~(size_t)1);
        if (COMP) smem += sizeof(double) * T * threads;
        if (CURVED) smem += sizeof(double2) * W * 2 * RING_G * V + 16;   // coefficient staging (after the 16-byte aligned int tables)
        return smem;
    };
    // register budget: per-thread state is T x (3 + NSRC) + NSRC x V doubles; CTAs of <= 128 threads
    // are compiled for 3 co-resident CTAs per SM (168 registers) while that fits, else for 2
    // (the open-universe kernels also hold the tile's 2 V coefficients: 2 CTAs)
    constexpr int MINB128 = (CURVED || 2 * (T * (3 + NSRC) + NSRC * V) > 140) ? 2 : MINB_128;
    const bool small = sh.threads <= 128;
    // multi-pass launches always run 128 threads x T_MAX points (choose_shape): one more kernel, not 24
    const bool multi = sh.n_pass > 1;
    if (multi && !(T == T_MAX && small)) { set_error("internal: multi-pass shape %d x %d", sh.threads, T); return GCAMB_EINVAL; }
    void (*kern)(TransferParams) = small ? transfer_kernel<T, V, NSRC, RING_G, 128, MINB128, COMP, SPARSE, false, CURVED>
                                         : transfer_kernel<T, V, NSRC, RING_G, 256, MINB_256, COMP, SPARSE, false, CURVED>;
    if constexpr (T == T_MAX) {
        if (multi) kern = transfer_kernel<T, V, NSRC, RING_G, 128, MINB128, COMP, SPARSE, true, CURVED>;
    }
    // opt in to large dynamic shared memory once per kernel and device (bit d of the mask = device d done)
    static std::atomic<unsigned long long> attr_done[3];
    const int which = multi ? 2 : small;
    const unsigned long long dev_bit = 1ull << (device & 63);
    if (!(attr_done[which].load(std::memory_order_acquire) & dev_bit)) {
        GCAMB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)smem_bytes(small ? 128 : 256)));
        attr_done[which].fetch_or(dev_bit, std::memory_order_release);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(n_pos * prm.n_batch));
    cfg.blockDim = dim3((unsigned)sh.threads);
    cfg.dynamicSmemBytes = smem_bytes(small ? 128 : 256);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = overlap_previous ? 1 : 0;
    GCAMB_CUDA(cudaLaunchKernelEx(&cfg, kern, prm));
    return GCAMB_OK;
}

// Positions [pos0, pos1) of the cost order.  The first n_comp positions of the order (the largest
// k: x_max = k chi_0 above COMP_X_MIN) run the compensated body in a launch of their own, issued
// first because they are the heaviest rows; the plain launch follows, overlapped with it.
// `zero_fill`: this range also zeroes the skipped region of Delta (for all rows).
// SPARSE: the kernels that skip the accumulation on tiles without a listed l (sparse l lists).
template <int T, int V, int NSRC, bool SPARSE, bool CURVED>
static gcamb_status launch_pair(const TransferParams &prm, const TransferShape &sh, int n_comp, int pos0, int pos1,
                                bool zero_fill, int device, cudaStream_t stream)
{
    if constexpr (CURVED)   // one launch: the open-universe kernels have no compensated form (the plan sets n_comp = 0)
        return launch_impl<T, V, NSRC, false, false, true>(prm, sh, pos0, pos1 - pos0, zero_fill, false, device, stream);
    else {
    const int c0 = pos0, c1 = std::min(pos1, n_comp);   // compensated part
    const int q0 = std::max(pos0, n_comp), q1 = pos1;   // plain part
    const bool has_plain = q1 > q0;
    gcamb_status st = launch_impl<T, V, NSRC, true, SPARSE, false>(prm, sh, c0, c1 - c0, zero_fill && !has_plain, prm.overlap_prev != 0, device, stream);
    if (st != GCAMB_OK) return st;
    return launch_impl<T, V, NSRC, false, SPARSE, false>(prm, sh, q0, q1 - q0, zero_fill, c1 > c0 || prm.overlap_prev != 0, device, stream);
    }
}

template <int V, int NSRC, bool SPARSE, bool CURVED>
static gcamb_status launch_T(const TransferParams &prm, const TransferShape &sh, int n_comp, int pos0, int pos1,
                             bool zero_fill, int device, cudaStream_t stream)
{
    switch (sh.T) {
#define GCAMB_T(t) case t: return launch_pair<t, V, NSRC, SPARSE, CURVED>(prm, sh, n_comp, pos0, pos1, zero_fill, device, stream);
        GCAMB_T(1) GCAMB_T(2) GCAMB_T(3) GCAMB_T(4) GCAMB_T(5) GCAMB_T(6)
        GCAMB_T(7) GCAMB_T(8) GCAMB_T(9) GCAMB_T(10) GCAMB_T(11) GCAMB_T(12)
#undef GCAMB_T
    }
    set_error("no transfer kernel for T=%d", sh.T);
    return GCAMB_EINVAL;
}

// The kernel instantiations (12 T x 2 coefficient forms x 2 CTA sizes per entry) dominate the build,
// so build.py compiles this file once per entry below (-DGCAMB_TU_SPARSE=s
// -DGCAMB_TU_NSRC=n), in parallel; the host-side functions live in the (0, 2) unit.  Without the
// macros everything is one translation unit.
// Two more units (-DGCAMB_TU_CURVED=1 -DGCAMB_TU_NSRC=n) hold the open-universe kernels (dense only: a sparse
// l list is served by the dense kernels, which store the listed l only).
#ifdef GCAMB_TU_SPARSE
#ifndef GCAMB_TU_CURVED
#define GCAMB_TU_CURVED 0
#endif
#define GCAMB_TU_HAS(sp, ns) (!GCAMB_TU_CURVED && (sp) == GCAMB_TU_SPARSE && (ns) == GCAMB_TU_NSRC)
#define GCAMB_TU_HAS_CURVED(ns) (GCAMB_TU_CURVED && (ns) == GCAMB_TU_NSRC)
#define GCAMB_TU_PRIMARY (!GCAMB_TU_CURVED && GCAMB_TU_SPARSE == 0 && GCAMB_TU_NSRC == 2)
#else
#define GCAMB_TU_HAS(sp, ns) 1
#define GCAMB_TU_HAS_CURVED(ns) 1
#define GCAMB_TU_PRIMARY 1
#endif
#define GCAMB_ENTRY(name, NS, SP, CV)                                                                         \
    gcamb_status name(const TransferParams &prm, const TransferShape &sh, int n_comp, int pos0, int pos1,     \
                      bool zero_fill, int device, cudaStream_t stream)                                        \
    {                                                                                                         \
        return launch_T<TILE_V, NS, SP, CV>(prm, sh, n_comp, pos0, pos1, zero_fill, device, stream);          \
    }
gcamb_status launch_range_dense_2(const TransferParams &, const TransferShape &, int, int, int, bool, int, cudaStream_t);
gcamb_status launch_range_dense_3(const TransferParams &, const TransferShape &, int, int, int, bool, int, cudaStream_t);
gcamb_status launch_range_sparse_2(const TransferParams &, const TransferShape &, int, int, int, bool, int, cudaStream_t);
gcamb_status launch_range_sparse_3(const TransferParams &, const TransferShape &, int, int, int, bool, int, cudaStream_t);
gcamb_status launch_range_dense_4(const TransferParams &, const TransferShape &, int, int, int, bool, int, cudaStream_t);
gcamb_status launch_range_sparse_4(const TransferParams &, const TransferShape &, int, int, int, bool, int, cudaStream_t);
gcamb_status launch_range_curved_2(const TransferParams &, const TransferShape &, int, int, int, bool, int, cudaStream_t);
gcamb_status launch_range_curved_3(const TransferParams &, const TransferShape &, int, int, int, bool, int, cudaStream_t);
#if GCAMB_TU_HAS(0, 2)
GCAMB_ENTRY(launch_range_dense_2, 2, false, false)
#endif
#if GCAMB_TU_HAS(0, 3)
GCAMB_ENTRY(launch_range_dense_3, 3, false, false)
#endif
#if GCAMB_TU_HAS(1, 2)
GCAMB_ENTRY(launch_range_sparse_2, 2, true, false)
#endif
#if GCAMB_TU_HAS(1, 3)
GCAMB_ENTRY(launch_range_sparse_3, 3, true, false)
#endif
#if GCAMB_TU_HAS(0, 4)
GCAMB_ENTRY(launch_range_dense_4, 4, false, false)
#endif
#if GCAMB_TU_HAS(1, 4)
GCAMB_ENTRY(launch_range_sparse_4, 4, true, false)
#endif
#if GCAMB_TU_HAS_CURVED(2)
GCAMB_ENTRY(launch_range_curved_2, 2, false, true)
#endif
#if GCAMB_TU_HAS_CURVED(3)
GCAMB_ENTRY(launch_range_curved_3, 3, false, true)
#endif

#if GCAMB_TU_PRIMARY
int transfer_tile_v() { return TILE_V; }

gcamb_status launch_transfer(const gcamb_los_plan *p, int n_batch, const double *S_T,
                             const double *S_E, const double *S_phi, double *Delta,
                             cudaStream_t stream)
{
    return launch_transfer_range(p, n_batch, S_T, S_E, S_phi, Delta, 0, p->n_k, true, stream);
}

// S_4 != NULL: the four-sum kernels (tensor plans, tensor.cu)
static gcamb_status launch_range_any(const gcamb_los_plan *p, int n_batch, const double *S_T,
                                     const double *S_E, const double *S_phi, const double *S_4, double *Delta,
                                     int pos0, int pos1, bool zero_fill, cudaStream_t stream,
                                     const TransferShape *shape = nullptr, bool overlap_prev = false)
{
    const TransferShape &sh = shape ? *shape : p->shape;
    TransferParams prm;
    prm.overlap_prev = overlap_prev;
    prm.S[0] = S_T; prm.S[1] = S_E; prm.S[2] = S_phi; prm.S[3] = S_4;
    prm.Delta = Delta;
    prm.k = p->d_k; prm.chi = p->d_chi; prm.w = p->d_w; prm.pref = p->d_pref; prm.inv_x = p->d_inv;
    prm.start = p->d_start; prm.tile = p->d_tile; prm.korder = p->d_korder; prm.l_index = p->d_l_index;
    prm.l_list = p->d_l_list; prm.kz = p->d_kz; prm.tile_mask = p->d_tile_mask;
    prm.n_k = p->n_k; prm.n_tau = p->n_tau; prm.n_l = p->n_l;
    prm.l_min = p->l_min; prm.l_max = p->l_max; prm.n_tiles = p->n_tiles;
    prm.n_batch = n_batch; prm.n_pass = sh.n_pass; prm.pass_len = sh.pass_len;
    prm.l_contig = p->n_l == p->l_max - p->l_min + 1;
    prm.order_reversed = p->order_reversed;
    prm.cth = p->d_cth; prm.s2 = p->d_s2; prm.ib2 = p->d_ib2; prm.coef = p->d_coef; prm.l_end = p->d_l_end;
    if (p->curved)
        return (p->n_src_walk == 2 ? launch_range_curved_2 : launch_range_curved_3)(prm, sh, 0, pos0, pos1, zero_fill, p->device, stream);
    const bool sparse = p->d_tile_mask != nullptr;   // some tile holds no listed l
    if (S_4) return (sparse ? launch_range_sparse_4 : launch_range_dense_4)(prm, sh, p->n_comp, pos0, pos1, zero_fill, p->device, stream);
    if (p->n_src_walk == 2)
        return (sparse ? launch_range_sparse_2 : launch_range_dense_2)(prm, sh, p->n_comp, pos0, pos1, zero_fill, p->device, stream);
    return (sparse ? launch_range_sparse_3 : launch_range_dense_3)(prm, sh, p->n_comp, pos0, pos1, zero_fill, p->device, stream);
}

gcamb_status launch_transfer_range(const gcamb_los_plan *p, int n_batch, const double *S_T,
                                   const double *S_E, const double *S_phi, double *Delta,
                                   int pos0, int pos1, bool zero_fill, cudaStream_t stream)
{
    return launch_range_any(p, n_batch, S_T, S_E, S_phi, nullptr, Delta, pos0, pos1, zero_fill, stream);
}

gcamb_status launch_transfer4(const gcamb_los_plan *p, int n_batch, const double *S_0, const double *S_1,
                              const double *S_2, const double *S_3, double *Delta, cudaStream_t stream)
{
    if (p->curved || !S_3) { set_error("internal: four-sum kernels on a curved plan"); return GCAMB_EINVAL; }
    const TransferShape &sh = p->shape;
    // One pass of 128 threads with more than 5 points per thread: the four-sum kernels hold 254 registers, two thread
    // blocks of 4 warps per SM, and a launch of ~1000 rows ends on its few heaviest rows (the heaviest is 3/4 of an
    // SM's share at the paper's tensor sizes: SMs active for 82 % of the launch).  The first n_sm / 16 positions of
    // the cost order therefore run as thread blocks of 256 threads (a row done in half the time) in a launch of their
    // own, which the launch of the other rows overlaps (programmatic stream serialization, as behind the compensated
    // rows): 0.295 -> 0.254 ms; 32 such rows 0.260, 100 rows 0.277 ms (profiles/README.md 6.6).  The split depends
    // on the plan only, so a batched call and a single call still agree bit for bit.
    const int n_heavy = p->n_sm / 16;
    if (n_heavy > 0 && sh.n_pass == 1 && sh.threads == 128 && sh.T > 5 && 4 * n_heavy < p->n_k) {
        TransferShape big = sh;
        big.threads = 256;
        big.T = (p->n_tau + 255) / 256;
        gcamb_status st = launch_range_any(p, n_batch, S_0, S_1, S_2, S_3, Delta, 0, n_heavy, false, stream, &big, false);
        if (st != GCAMB_OK) return st;
        return launch_range_any(p, n_batch, S_0, S_1, S_2, S_3, Delta, n_heavy, p->n_k, true, stream, nullptr, true);
    }
    return launch_range_any(p, n_batch, S_0, S_1, S_2, S_3, Delta, 0, p->n_k, true, stream);
}
#endif   // GCAMB_TU_PRIMARY

}  // namespace gcamb
