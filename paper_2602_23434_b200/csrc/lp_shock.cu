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

    double ec[M], de[M];
#pragma unroll
    for (int i = 0; i < M; ++i) {
        ec[i] = __dsqrt_rn(__dmul_rn(tab[b0 + i], tab[b0 + i + 1]));      // geometric centre
        de[i] = active ? tab[(NB + 1) + b0 + i] : 0.0;                      // idle lanes (16 bins) weigh nothing
    }

    const long long gw = ((long long)blockIdx.x * kThreads + threadIdx.x) >> 5;
    const long long nw = ((long long)gridDim.x * kThreads) >> 5;
    for (long long p = gw; p < np; p += nw) {
        const double rr = r[p];
        if (!(rr > 1.0)) continue;                                          // no shock (warp-uniform)
        const double q = __dadd_rn(__ddiv_rn(__dmul_rn(3.0, rr), __dsub_rn(rr, 1.0)), q_r);   // Eq. 8
        double *row = chi + p * NB + b0;
        double c[M], term[M], t[M];
        double total = 0.0, n_in = 0.0;
#pragma unroll
        for (int i = 0; i < M; ++i) {
            c[i] = active ? row[i] : 0.0;
            term[i] = c[i] * pow(ec[i], q - 3.0) * de[i];
            total += term[i];
            n_in = fma(c[i], de[i], n_in);
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
            t[i] = pow(ec[i], 2.0 - q) * (below + 0.5 * term[i]);
            below += term[i];
            n_out = fma(t[i], de[i], n_out);
        }
        n_in = warp_sum(n_in);
        n_out = warp_sum(n_out);
        if (n_out != 0.0 && n_out == n_out) {                               // else: leave the row (S4)
            const double norm = n_in / n_out;
            if (active) {
#pragma unroll
                for (int i = 0; i < M; ++i) row[i] = norm * t[i];
            }
        }
    }
}

template <int NB>
int launch(const double *tab, const double *r, double q_r, double *chi, long long np, int sm_count, cudaStream_t s)
{
    long long blocks = (np + kWarps - 1) / kWarps;
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
