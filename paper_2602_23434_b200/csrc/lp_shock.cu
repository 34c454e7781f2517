// lp_shock.cu -- spectrum of the particles that cross a shock (Eq. 7-8; readings S1-S4
// of DESIGN.md section 3):
//   chi_out,i = C ec_i^(2-q) [ sum_{j<i} chi_j ec_j^(q-3) dE_j + (1/2) chi_i ec_i^(q-3) dE_i ],
//   q = 3r/(r-1) + q_R,   C from number conservation,   ec_i = sqrt(E_i E_{i+1}).
// The integral of Eq. 7 is a weighted prefix sum over the bins: a group of G lanes per flagged row, M
// contiguous bins per lane, a lane-local running sum plus an exclusive scan of the lane totals over the group
// (SHFL.UP), two group reductions for the normalisation.  Rows with r <= 1 (or NaN) are not touched and
// cost 8 bytes.  sm_100a.
#include "lp_device.cuh"

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

// A row is held by G = N_b/M lanes, M contiguous bins per lane (M = 4 up to 128 bins, then N_b/32), so a warp
// works on 32/G flagged rows at once -- at 64 bins two rows share the warp's instructions, at 16 bins eight.
template <int NB>
struct LpShockCfg {
    static constexpr int M = NB >= 128 ? NB / 32 : 4;
    static constexpr int G = NB / M;
    static constexpr int PPW = 32 / G;
};

// Per-lane slice of the bin table: the M bins [sub*M, sub*M + M).
template <int M>
struct LpShockTab {
    double rec[M], de[M];      // 1/ec_i (ec = geometric bin centre), dE_i
    double lnec0;              // ln ec of the lane's first bin
    double dln;                // ln(ec_{i+1}/ec_i): the same for every bin of a log-spaced table
};

// One row per lane group (all 32 lanes call).  ec^(q-3) is a geometric sequence along the bins of a log-spaced
// table: one exp for the lane's first bin and one for the ratio replace an exp per bin, and
// ec^(2-q) = 1/(ec^(q-3) ec) comes from the reciprocal sequence -- two exp and two divisions per lane and row
// instead of one of each per bin (with those the kernel was bound by this arithmetic, not by HBM).  The table's
// rounding makes the sequence geometric to ~1e-15 in the exponent and the products accumulate to ~1e-13
// relative, far inside the 1e-10 parity bound.  Returns whether the row was changed (reading S4).
template <int M, int G>
__device__ __forceinline__ bool lp_shock_row(const LpShockTab<M> &tb, double rr, double q_r, double (&c)[M], int sub)
{
    const double q = __dadd_rn(__ddiv_rn(__dmul_rn(3.0, rr), __dsub_rn(rr, 1.0)), q_r);   // Eq. 8
    const double s3 = q - 3.0;
    const double rho = exp(s3 * tb.dln), irho = 1.0 / rho;
    double pw = exp(s3 * tb.lnec0), ipw = 1.0 / pw;                 // ec^(q-3) of the lane's first bin, and 1 / it
    double term[M], scale[M];
    double total = 0.0, n_in = 0.0;
#pragma unroll
    for (int i = 0; i < M; ++i) {
        term[i] = c[i] * pw * tb.de[i];
        scale[i] = ipw * tb.rec[i];                                 // ec^(2-q)
        total += term[i];
        n_in = fma(c[i], tb.de[i], n_in);
        pw *= rho;
        ipw *= irho;
    }
    // exclusive scan of the lane totals over the row's G lanes: what lies in the bins below this lane's
    double incl = total;
#pragma unroll
    for (int o = 1; o < G; o <<= 1) {
        const double u = __shfl_up_sync(kFull, incl, o, G);
        if (sub >= o) incl += u;
    }
    // (not incl - total: the lane's own total can exceed what lies below it by many orders of magnitude, and the
    // difference would lose exactly the digits the lane's first bins need)
    double below = __shfl_up_sync(kFull, incl, 1, G);
    if (sub == 0) below = 0.0;
    double n_out = 0.0;
    double t[M];
#pragma unroll
    for (int i = 0; i < M; ++i) {
        t[i] = (below + 0.5 * term[i]) * scale[i];
        below += term[i];
        n_out = fma(t[i], tb.de[i], n_out);
    }
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) {
        n_in += __shfl_xor_sync(kFull, n_in, o);
        n_out += __shfl_xor_sync(kFull, n_out, o);
    }
    const bool changed = n_out != 0.0 && n_out == n_out;            // else: leave the row (S4)
    if (changed) {
        const double norm = n_in / n_out;
#pragma unroll
        for (int i = 0; i < M; ++i) c[i] = norm * t[i];
    }
    return changed;
}

// The same on a per-particle energy grid (moving grid): the row's own edges e[0..M] (e[M] = the next lane's first
// edge or the top edge) give its centres and widths; nothing is geometric any more, so ec^(q-3) costs a log and an
// exp per bin.
template <int M, int G>
__device__ __forceinline__ bool lp_shock_row_grid(const double (&e)[M + 1], double rr, double q_r, double (&c)[M], int sub)
{
    const double q = __dadd_rn(__ddiv_rn(__dmul_rn(3.0, rr), __dsub_rn(rr, 1.0)), q_r);   // Eq. 8
    const double s3 = q - 3.0;
    double term[M], scale[M], de[M];
    double total = 0.0, n_in = 0.0;
#pragma unroll
    for (int i = 0; i < M; ++i) {
        const double ec = __dsqrt_rn(__dmul_rn(e[i], e[i + 1]));
        de[i] = __dsub_rn(e[i + 1], e[i]);
        const double pw = exp(s3 * log(ec));
        term[i] = c[i] * pw * de[i];
        scale[i] = 1.0 / (pw * ec);
        total += term[i];
        n_in = fma(c[i], de[i], n_in);
    }
    double incl = total;
#pragma unroll
    for (int o = 1; o < G; o <<= 1) {
        const double u = __shfl_up_sync(kFull, incl, o, G);
        if (sub >= o) incl += u;
    }
    double below = __shfl_up_sync(kFull, incl, 1, G);
    if (sub == 0) below = 0.0;
    double n_out = 0.0;
    double t[M];
#pragma unroll
    for (int i = 0; i < M; ++i) {
        t[i] = (below + 0.5 * term[i]) * scale[i];
        below += term[i];
        n_out = fma(t[i], de[i], n_out);
    }
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) {
        n_in += __shfl_xor_sync(kFull, n_in, o);
        n_out += __shfl_xor_sync(kFull, n_out, o);
    }
    const bool changed = n_out != 0.0 && n_out == n_out;
    if (changed) {
        const double norm = n_in / n_out;
#pragma unroll
        for (int i = 0; i < M; ++i) c[i] = norm * t[i];
    }
    return changed;
}

// one lane group per flagged row, plain 8-byte accesses (grid rows are 8-byte aligned only)
template <int NB>
__global__ void __launch_bounds__(kThreads)
lp_shock_grid_kernel(const double *__restrict__ eng, const double *__restrict__ r, double q_r,
                     double *__restrict__ chi, long long np)
{
    using C = LpShockCfg<NB>;
    constexpr int M = C::M, G = C::G, PPW = C::PPW;
    const int lane = threadIdx.x & 31;
    const int sub = lane % G, grp = lane / G;
    const int b0 = sub * M;
    const long long gw = ((long long)blockIdx.x * kThreads + threadIdx.x) >> 5;
    const long long nw = ((long long)gridDim.x * kThreads) >> 5;
    for (long long base = gw << 5; base < np; base += nw << 5) {
        const double r_lane = base + lane < np ? r[base + lane] : 0.0;
        const unsigned todo = __ballot_sync(kFull, r_lane > 1.0);
        const int nflag = __popc(todo);
        for (int k = 0; k < nflag; k += PPW) {
            const int idx = k + grp;
            const bool valid = idx < nflag;
            const int j = valid ? (int)__fns(todo, 0, idx + 1) : 0;
            const double rr = __shfl_sync(kFull, r_lane, j);
            double *row = chi + (base + j) * NB + b0;
            const double *er = eng + (base + j) * (NB + 1) + b0;
            double c[M], e[M + 1];
#pragma unroll
            for (int i = 0; i < M; ++i) {
                c[i] = valid ? row[i] : 0.0;
                e[i] = valid ? er[i] : 1.0 + i;
            }
            e[M] = valid ? er[M] : 1.0 + M;
            const bool changed = lp_shock_row_grid<M, G>(e, valid ? rr : 2.0, q_r, c, sub);
            if (valid && changed) {
#pragma unroll
                for (int i = 0; i < M; ++i) row[i] = c[i];
            }
        }
    }
}

template <int NB>
__global__ void __launch_bounds__(kThreads)
lp_shock_kernel(const double *__restrict__ tab, const double *__restrict__ r, double q_r,
                double *__restrict__ chi, long long np)
{
    using C = LpShockCfg<NB>;
    constexpr int M = C::M, G = C::G, PPW = C::PPW;
    constexpr bool kStaged = M >= 8;              // rows through the transposing stage buffer (then G = 32, PPW = 1)
    __shared__ __align__(16) unsigned char sStage[kWarps][kStaged ? LpStage<M>::kBytes : 16];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane % G, grp = lane / G;
    const int b0 = sub * M;

    LpShockTab<M> tb;
#pragma unroll
    for (int i = 0; i < M; ++i) {
        const double ec = __dsqrt_rn(__dmul_rn(tab[b0 + i], tab[b0 + i + 1]));      // geometric centre
        tb.rec[i] = 1.0 / ec;
        tb.de[i] = tab[(NB + 1) + b0 + i];
        if (i == 0) tb.lnec0 = log(ec);
    }
    tb.dln = (log(tab[NB]) - log(tab[0])) / (double)NB;

    // a warp takes 32 consecutive particles at a time: one coalesced read of their r, a ballot of the flagged
    // ones, then the flagged rows PPW at a time -- unflagged particles cost their 8 bytes only
    const long long gw = ((long long)blockIdx.x * kThreads + threadIdx.x) >> 5;
    const long long nw = ((long long)gridDim.x * kThreads) >> 5;
    for (long long base = gw << 5; base < np; base += nw << 5) {
        const double r_lane = base + lane < np ? r[base + lane] : 0.0;
        const unsigned todo = __ballot_sync(kFull, r_lane > 1.0);                   // r <= 1 or NaN: no shock
        const int nflag = __popc(todo);
        for (int k = 0; k < nflag; k += PPW) {
            const int idx = k + grp;                                                // this group's flagged row
            const bool valid = idx < nflag;
            const int j = valid ? (int)__fns(todo, 0, idx + 1) : 0;                // the idx-th set bit of todo
            const double rr = __shfl_sync(kFull, r_lane, j);
            double *row = chi + (base + j) * NB;
            double c[M];
            if constexpr (kStaged) {
                double2 t2[M / 2];
                LpStage<M>::fetch(row, lane, t2);                                   // (valid is warp-uniform: PPW = 1)
                LpStage<M>::place(t2, sStage[warp], lane, c);
            } else {
#pragma unroll
                for (int i = 0; i < M; i += 2) {
                    const double2 v = valid ? *reinterpret_cast<const double2 *>(row + b0 + i) : make_double2(0.0, 0.0);
                    c[i] = v.x;
                    c[i + 1] = v.y;
                }
            }
            const bool changed = lp_shock_row<M, G>(tb, valid ? rr : 2.0, q_r, c, sub);
            if constexpr (kStaged) {
                if (changed) LpStage<M>::store(row, sStage[warp], lane, c);         // (uniform over the warp)
            } else if (valid && changed) {
#pragma unroll
                for (int i = 0; i < M; i += 2) *reinterpret_cast<double2 *>(row + b0 + i) = make_double2(c[i], c[i + 1]);
            }
        }
    }
}

template <int NB>
int launch(const double *tab, const double *eng, const double *r, double q_r, double *chi, long long np, int sm_count,
           cudaStream_t s)
{
    long long blocks = (np + kWarps * 32 - 1) / (kWarps * 32);          // a warp takes 32 particles per trip
    const long long cap = (long long)sm_count * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    if (eng) lp_shock_grid_kernel<NB><<<(int)blocks, kThreads, 0, s>>>(eng, r, q_r, chi, np);
    else lp_shock_kernel<NB><<<(int)blocks, kThreads, 0, s>>>(tab, r, q_r, chi, np);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace

int lp_launch_shock(const double *tab, const double *eng, const double *r, double q_r, double *chi, long long np,
                    int nbins, int sm_count, cudaStream_t s)
{
    switch (nbins) {
    case 16:  return launch<16>(tab, eng, r, q_r, chi, np, sm_count, s);
    case 32:  return launch<32>(tab, eng, r, q_r, chi, np, sm_count, s);
    case 64:  return launch<64>(tab, eng, r, q_r, chi, np, sm_count, s);
    case 128: return launch<128>(tab, eng, r, q_r, chi, np, sm_count, s);
    case 256: return launch<256>(tab, eng, r, q_r, chi, np, sm_count, s);
    case 512: return launch<512>(tab, eng, r, q_r, chi, np, sm_count, s);
    default:  return -1;
    }
}
