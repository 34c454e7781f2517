// lp_shock.cu -- spectrum of the particles that cross a shock (Eq. 7-8; readings S1-S4
// of DESIGN.md section 3):
//   chi_out,i = C ec_i^(2-q) [ sum_{j<i} chi_j ec_j^(q-3) dE_j + (1/2) chi_i ec_i^(q-3) dE_i ],
//   q = 3r/(r-1) + q_R,   C from number conservation,   ec_i = sqrt(E_i E_{i+1}).
// The integral of Eq. 7 is a weighted prefix sum over the bins: one warp per flagged row, M = N_b/32
// contiguous bins per lane, a lane-local running sum plus an exclusive warp scan of the lane totals
// (SHFL.UP), two warp reductions for the normalisation.  Rows with r <= 1 (or NaN) are not touched and
// cost 8 bytes.  sm_100a.
#include "lp_internal.h"

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}

// Per-lane slice of the bin table for the shock update: M contiguous bins of lane `lane`.
template <int M>
struct LpShockTab {
    double ec[M], lnec[M], de[M];
};

// One flagged row, all 32 lanes.  ec^(q-3) = exp((q-3) ln ec) with ln ec tabulated per lane, and
// ec^(2-q) = 1 / (ec^(q-3) ec): one exp and one division per bin and row instead of two pow (the kernel is
// bound by this arithmetic, not by HBM); relative error ~ |q-3| ln(ec) ulp ~ 1e-14, far inside the 1e-10
// parity bound.
template <int M>
__device__ __forceinline__ void lp_shock_row(const LpShockTab<M> &tb, double rr, double q_r, double *row,
                                             bool active, int lane)
{
    const double q = __dadd_rn(__ddiv_rn(__dmul_rn(3.0, rr), __dsub_rn(rr, 1.0)), q_r);   // Eq. 8
    const double s3 = q - 3.0;
    double c[M], term[M], t[M], pw[M];
    double total = 0.0, n_in = 0.0;
#pragma unroll
    for (int i = 0; i < M; ++i) {
        c[i] = active ? row[i] : 0.0;
        pw[i] = exp(s3 * tb.lnec[i]);                                       // ec^(q-3)
        term[i] = c[i] * pw[i] * tb.de[i];
        total += term[i];
        n_in = fma(c[i], tb.de[i], n_in);
    }
    // exclusive scan of the lane totals: what lies in the bins below this lane's
    double incl = total;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double u = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += u;
    }
    double below = incl - total;
    double n_out = 0.0;
#pragma unroll
    for (int i = 0; i < M; ++i) {
        t[i] = (below + 0.5 * term[i]) / (pw[i] * tb.ec[i]);                // ec^(2-q) = 1 / (ec^(q-3) ec)
        below += term[i];
        n_out = fma(t[i], tb.de[i], n_out);
    }
    n_in = warp_sum(n_in);
    n_out = warp_sum(n_out);
    if (n_out != 0.0 && n_out == n_out) {                                   // else: leave the row (S4)
        const double norm = n_in / n_out;
        if (active) {
#pragma unroll
            for (int i = 0; i < M; ++i) row[i] = norm * t[i];
        }
    }
}

template <int NB>
__global__ void __launch_bounds__(kThreads)
lp_shock_kernel(const double *__restrict__ tab, const double *__restrict__ r, double q_r,
                double *__restrict__ chi, long long np)
{
    constexpr int M = NB >= 32 ? NB / 32 : 1;          // bins per lane
    constexpr int LANES = NB >= 32 ? 32 : NB;          // lanes that hold bins (16 bins: half a warp)
    const int lane = threadIdx.x & 31;
    const bool active = lane < LANES;
    const int b0 = active ? lane * M : 0;

    LpShockTab<M> tb;
#pragma unroll
    for (int i = 0; i < M; ++i) {
        tb.ec[i] = __dsqrt_rn(__dmul_rn(tab[b0 + i], tab[b0 + i + 1]));    // geometric centre
        tb.lnec[i] = log(tb.ec[i]);
        tb.de[i] = active ? tab[(NB + 1) + b0 + i] : 0.0;                   // idle lanes (16 bins) weigh nothing
    }

    // a warp takes 32 consecutive particles at a time: one coalesced read of their r, a ballot of the
    // flagged ones, then one flagged row after the other -- unflagged particles cost their 8 bytes only
    const long long gw = ((long long)blockIdx.x * kThreads + threadIdx.x) >> 5;
    const long long nw = ((long long)gridDim.x * kThreads) >> 5;
    for (long long base = gw << 5; base < np; base += nw << 5) {
        const double r_lane = base + lane < np ? r[base + lane] : 0.0;
        unsigned todo = __ballot_sync(kFull, r_lane > 1.0);                 // r <= 1 or NaN: no shock
        while (todo) {
            const int j = __ffs(todo) - 1;
            todo &= todo - 1;
            lp_shock_row<M>(tb, __shfl_sync(kFull, r_lane, j), q_r, chi + (base + j) * NB + b0, active, lane);
        }
    }
}

template <int NB>
int launch(const double *tab, const double *r, double q_r, double *chi, long long np, int sm_count, cudaStream_t s)
{
    long long blocks = (np + kWarps * 32 - 1) / (kWarps * 32);          // a warp takes 32 particles per trip
    const long long cap = (long long)sm_count * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    lp_shock_kernel<NB><<<(int)blocks, kThreads, 0, s>>>(tab, r, q_r, chi, np);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace

int lp_launch_shock(const double *tab, const double *r, double q_r, double *chi, long long np, int nbins,
                    int sm_count, cudaStream_t s)
{
    switch (nbins) {
    case 16:  return launch<16>(tab, r, q_r, chi, np, sm_count, s);
    case 32:  return launch<32>(tab, r, q_r, chi, np, sm_count, s);
    case 64:  return launch<64>(tab, r, q_r, chi, np, sm_count, s);
    case 128: return launch<128>(tab, r, q_r, chi, np, sm_count, s);
    case 256: return launch<256>(tab, r, q_r, chi, np, sm_count, s);
    case 512: return launch<512>(tab, r, q_r, chi, np, sm_count, s);
    default:  return -1;
    }
}
