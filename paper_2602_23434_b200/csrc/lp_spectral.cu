// lp_spectral.cu -- spectral update of every particle (steps a7-a10 of DESIGN.md section 1):
// coefficients and CFL substep count thread-per-particle, then the donor-cell upwind substeps
// with the row's N_b bins spread over the lanes of a warp and kept in registers.
// Solves Eq. 6 of the paper with the loss term of Eq. 4.  sm_100a.
#include "lp_device.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr unsigned kFull = 0xffffffffu;

struct __align__(16) LpCoef {      // per-particle scalars handed from phase 1 to phase 2
    double a;      // (1/3) div_mu u^mu
    double cr;     // c_r
    double dts;    // dtau / n_sub
    int ns;        // n_sub (0 = no particle)
    int pad;
};

// Phase 1 (one thread = one particle): gather v, B, rho at x^{n+1}; gamma_g, dtau, c_r, a
// (PAPER.md:85, 96-99, 105); lambda = max_i outflow rate of bin i; n_sub = ceil(dtau*lambda/C_E).
template <int NB>
__device__ __forceinline__ void lp_phase1(const LpSpectralArgs &A, long long p, const double *sE,
                                          const double *sR, LpCoef &c, int &ns_signed)
{
    LpStencil st;
    lp_stencil(A.g, A.x[p], A.y[p], A.z[p], st);
    double qa[4], qb[3];
    lp_gather_A(A.cells, st, qa);
    lp_gather_B(A.cells, st, qb);
    const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(qa[0], qa[0]), __dmul_rn(qa[1], qa[1])), __dmul_rn(qa[2], qa[2]));
    const double b2 = __dadd_rn(__dadd_rn(__dmul_rn(qb[0], qb[0]), __dmul_rn(qb[1], qb[1])), __dmul_rn(qb[2], qb[2]));
    const double gam = __ddiv_rn(1.0, __dsqrt_rn(__dsub_rn(1.0, v2)));
    const double dtau = __ddiv_rn(A.dt, gam);
    const double cr = __dmul_rn(A.kappa, __dadd_rn(__dmul_rn(0.5, b2), A.u_rad));
    const double a = __ddiv_rn(-log(__ddiv_rn(qa[3], A.rho_old[p])), __dmul_rn(3.0, dtau));

    double lam = 0.0;
    double e0 = sE[0];
    double wl = -e0 * fma(cr, e0, a);
#pragma unroll 8
    for (int i = 0; i < NB; ++i) {
        const double e = sE[i + 1];
        const double wr = -e * fma(cr, e, a);
        const double out = (fmax(wr, 0.0) - fmin(wl, 0.0)) * sR[i];
        lam = fmax(lam, out);
        wl = wr;
    }
    const double need = ceil(__ddiv_rn(__dmul_rn(dtau, lam), A.cfl_e));
    int n = !(need >= 1.0) ? 1 : (need > 2.0e9 ? 2000000000 : (int)need);
    const bool capped = n > A.max_substeps;
    if (capped) n = A.max_substeps;
    c.a = a;
    c.cr = cr;
    c.dts = __ddiv_rn(dtau, (double)n);
    c.ns = n;
    c.pad = 0;
    ns_signed = capped ? -n : n;
}

template <int M>
__device__ __forceinline__ void lp_load_row(const double *__restrict__ src, double (&v)[M])
{
    if constexpr (M == 1) {
        v[0] = *src;
    } else {
#pragma unroll
        for (int i = 0; i < M; i += 2) {
            double2 t = *reinterpret_cast<const double2 *>(src + i);
            v[i] = t.x;
            v[i + 1] = t.y;
        }
    }
}

template <int M>
__device__ __forceinline__ void lp_store_row(double *__restrict__ dst, const double (&v)[M])
{
    if constexpr (M == 1) {
        *dst = v[0];
    } else {
#pragma unroll
        for (int i = 0; i < M; i += 2) *reinterpret_cast<double2 *>(dst + i) = make_double2(v[i], v[i + 1]);
    }
}

// Phase 2 for one row held as M bins per lane over G lanes.  Donor-cell upwind:
//   chi_i <- chi_i - c_i (F_{i+1} - F_i),  F_k = w_k * (w_k > 0 ? chi_{k-1} : chi_k),  chi_{-1} = chi_{Nb} = 0
// evaluated as two FMAs per bin with alpha_i = c_i w_i, beta_i = c_i w_{i+1}.
template <int M, int G, bool DIAG>
__device__ __forceinline__ void lp_row_substeps(double (&chi)[M], const double *eE, const double *eR,
                                                const LpCoef &c, int nloop, int sub, double &lost)
{
    double al[M], be[M];
    bool pos[M + 1];
    double w_first, w_last;
    {
        double wprev = -eE[0] * fma(c.cr, eE[0], c.a);
        w_first = wprev;
        pos[0] = wprev > 0.0;
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const double e = eE[i + 1];
            const double wn = -e * fma(c.cr, e, c.a);
            const double ci = c.dts * eR[i];
            al[i] = ci * wprev;
            be[i] = ci * wn;
            pos[i + 1] = wn > 0.0;
            wprev = wn;
        }
        w_last = wprev;
    }
    double s0 = 0.0, s1 = 0.0;
    for (int s = 0; s < nloop; ++s) {
        double left = __shfl_up_sync(kFull, chi[M - 1], 1, G);
        double right = __shfl_down_sync(kFull, chi[0], 1, G);
        if (sub == 0) left = 0.0;
        if (sub == G - 1) right = 0.0;
        if (s < c.ns) {
            if (DIAG) { s0 += chi[0]; s1 += chi[M - 1]; }
            double d[M + 1];
            d[0] = pos[0] ? left : chi[0];
#pragma unroll
            for (int i = 1; i < M; ++i) d[i] = pos[i] ? chi[i - 1] : chi[i];
            d[M] = pos[M] ? chi[M - 1] : right;
#pragma unroll
            for (int i = 0; i < M; ++i) chi[i] = fma(al[i], d[i], fma(-be[i], d[i + 1], chi[i]));
        }
    }
    if (DIAG) {
        double t1 = (sub == G - 1) ? fmax(w_last, 0.0) * s1 : 0.0;
        double t0 = (sub == 0) ? fmin(w_first, 0.0) * s0 : 0.0;
        t1 = __shfl_sync(kFull, t1, G - 1, G);
        t0 = __shfl_sync(kFull, t0, 0, G);
        lost = c.dts * (t1 - t0);
    }
}

template <int NB, bool DIAG>
__global__ void __launch_bounds__(kThreads) lp_spectral_kernel(LpSpectralArgs A)
{
    constexpr int G = NB >= 32 ? 32 : NB;     // lanes that share one row
    constexpr int M = NB / G;                 // bins per lane (contiguous)
    constexpr int PPW = 32 / G;               // rows a warp works on at once
    constexpr int ROWS = 32 / PPW;            // row iterations per chunk of 32 particles
    constexpr int U = (M <= 2) ? 4 : (M == 4 ? 2 : 1);   // rows in flight per warp
    constexpr bool kTabInRegs = (M <= 4);

    __shared__ __align__(16) double sE[NB + 2];
    __shared__ __align__(16) double sR[NB];
    __shared__ LpCoef sC[kWarps][32];

    for (int i = threadIdx.x; i <= NB; i += kThreads) sE[i] = A.tab[i];
    for (int i = threadIdx.x; i < NB; i += kThreads) sR[i] = A.tab[(NB + 1) + NB + i];
    __syncthreads();

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane % G, grp = lane / G;

    double rE[kTabInRegs ? M + 1 : 1], rR[kTabInRegs ? M : 1];
    if (kTabInRegs) {
#pragma unroll
        for (int i = 0; i <= M; ++i) rE[i] = sE[sub * M + i];
#pragma unroll
        for (int i = 0; i < M; ++i) rR[i] = sR[sub * M + i];
    }
    const double *eE = kTabInRegs ? rE : (sE + sub * M);
    const double *eR = kTabInRegs ? rR : (sR + sub * M);

    const long long nchunks = (A.np + 31) >> 5;
    const long long gw = (long long)blockIdx.x * kWarps + warp;
    const long long nw = (long long)gridDim.x * kWarps;

    for (long long chunk = gw; chunk < nchunks; chunk += nw) {
        const long long base = chunk << 5;
        {   // ---- phase 1: lane <-> particle base + lane
            const long long p = base + lane;
            LpCoef c;
            c.a = 0.0; c.cr = 0.0; c.dts = 0.0; c.ns = 0; c.pad = 0;
            if (p < A.np) {
                int nss;
                lp_phase1<NB>(A, p, sE, sR, c, nss);
                A.nsub_ws[p] = nss;
                if (A.nsub_user) A.nsub_user[p] = nss;
            }
            sC[warp][lane] = c;
        }
        __syncwarp();
        // ---- phase 2: rows of the chunk, PPW at a time, U loads in flight
        for (int j0 = 0; j0 < ROWS; j0 += U) {
            double buf[U][M];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const long long pj = base + (j0 + u) * PPW + grp;
                if (pj < A.np) lp_load_row<M>(A.chi_in + pj * NB + sub * M, buf[u]);
                else {
#pragma unroll
                    for (int i = 0; i < M; ++i) buf[u][i] = 0.0;
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int r = (j0 + u) * PPW + grp;
                const long long pj = base + r;
                const LpCoef c = sC[warp][r];
                int nloop = c.ns;
                if (PPW > 1) nloop = max(nloop, __shfl_xor_sync(kFull, nloop, 16));
                double lost = 0.0;
                lp_row_substeps<M, G, DIAG>(buf[u], eE, eR, c, nloop, sub, lost);
                if (pj < A.np) {
                    lp_store_row<M>(A.chi_out + pj * NB + sub * M, buf[u]);
                    if (DIAG && sub == 0) {
                        A.lost_ws[pj] = lost;
                        if (A.lost_user) A.lost_user[pj] = lost;
                    }
                }
            }
        }
        __syncwarp();
    }
}

template <int NB>
int launch_nb(const LpSpectralArgs &a, bool diag, int sm_count, cudaStream_t s)
{
    const long long nchunks = (a.np + 31) >> 5;
    long long want = (nchunks + kWarps - 1) / kWarps;
    int per_sm = 1;
    if (diag) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lp_spectral_kernel<NB, true>, kThreads, 0);
    else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lp_spectral_kernel<NB, false>, kThreads, 0);
    if (per_sm < 1) per_sm = 1;
    long long cap = (long long)sm_count * per_sm;
    int blocks = (int)(want < cap ? want : cap);
    if (blocks < 1) blocks = 1;
    if (diag) lp_spectral_kernel<NB, true><<<blocks, kThreads, 0, s>>>(a);
    else lp_spectral_kernel<NB, false><<<blocks, kThreads, 0, s>>>(a);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace

int lp_launch_spectral(const LpSpectralArgs &a, int nbins, bool diag, int sm_count, cudaStream_t s)
{
    switch (nbins) {
    case 16:  return launch_nb<16>(a, diag, sm_count, s);
    case 32:  return launch_nb<32>(a, diag, sm_count, s);
    case 64:  return launch_nb<64>(a, diag, sm_count, s);
    case 128: return launch_nb<128>(a, diag, sm_count, s);
    case 256: return launch_nb<256>(a, diag, sm_count, s);
    case 512: return launch_nb<512>(a, diag, sm_count, s);
    default:  return -1;
    }
}
