// lp_spectral.cu -- spectral update of every particle (steps a7-a10 of DESIGN.md section 1) and,
// when fused, the two push stages (a5, a6) in front of it.
//
// Phase 1 (one thread = one particle): [push 0, push 1,] gather v, B, rho at x^{n+1}, coefficients,
// CFL substep count.  Phase 2 (a group of G = N_b/M lanes = one row, M contiguous bins per lane in
// registers): n_sub donor-cell upwind substeps of Eq. 6 with the loss term of Eq. 4
// (PAPER.md:96); the only cross-lane traffic per substep is one shuffle up and one shuffle down.
//
// Two kernels:
//  * lp_spectral_bulk_kernel (N_b <= 256), warp-specialised: particle warps run phase 1 and hand the
//    coefficients through a shared-memory ring (mbarrier full/empty) to row warps, which stream the
//    rows through private rings of shared-memory slots filled and drained by the TMA engine
//    (cp.async.bulk + mbarrier).  Measured on B200: phase 1 is a chain of dependent gathers (latency)
//    and phase 2 a stream (HBM); run by the same warp one after the other their times add, run by
//    different warps they overlap.
//  * lp_spectral_direct_kernel (N_b = 512, 16 bins per lane): every warp does both phases; rows move with
//    coalesced accesses through a transposing staging buffer, one row fetched ahead.
// sm_100a.
#include "lp_device.cuh"

namespace {

constexpr unsigned kFull = 0xffffffffu;

// Per-particle scalars handed from phase 1 to phase 2.  The substeps only ever need the products
// (dtau/n_sub)/2 * a and (dtau/n_sub)/2 * c_r, so phase 1 (one thread per particle) forms them once.
struct LpCoef {
    double a2;     // (dts/2) * a,    a = (1/3) div_mu u^mu,   dts = dtau / n_sub
    double cr2;    // (dts/2) * c_r
    int ns;        // n_sub (0 = no particle)
    int cool;      // a + c_r E_0 >= 0: every edge velocity is <= 0 (LpRow::setup_cool)
};

// outflow rate of bin i:  (max(w_{i+1},0) - min(w_i,0)) / dE_i,   w_k = -E_k (a + c_r E_k)
__device__ __forceinline__ double lp_outflow(const double *sE, const double *sR, int i, double a, double cr)
{
    const double el = sE[i], er = sE[i + 1];
    const double wl = -el * fma(cr, el, a);
    const double wr = -er * fma(cr, er, a);
    return (fmax(wr, 0.0) - fmin(wl, 0.0)) * sR[i];
}

// Phase 1.  FUSED: the two push stages (same arithmetic as lp_push0/1_kernel)
// run first on the same thread, so k1, x*, rho_old never leave registers.
template <int NB, bool FUSED>
__device__ __forceinline__ void lp_phase1(const LpSpectralArgs &A, long long p, double px, double py, double pz,
                                          const double *sE, const double *sR, LpCoef &c, int &ns_signed)
{
    double a, cr, dtau;
    lp_particle_coefficients<FUSED>(A.g, A.cells, A.dt, A.kappa, A.u_rad, A.x, A.y, A.z, A.status, A.rho_old, p, px, py, pz,
                                    a, cr, dtau);

    // lambda = max_i outflow_i.  On the library's log-spaced table the maximum sits in the first or the
    // last bin up to the rounding noise of E/dE (LpLamCand::margin, >= 1e-12), so those two bins decide n_sub
    // unless dtau*lambda/C_E is within that margin of an integer; only then (practically never) are the other
    // hull-vertex bins (see LpLamCand) evaluated too.  The result is the same integer either way.
    auto cand_outflow = [&](int k) -> double {             // table values straight from the kernel parameters
        const double el = A.cand.el[k], er = A.cand.er[k];
        const double wl = -el * fma(cr, el, a);
        const double wr = -er * fma(cr, er, a);
        return (fmax(wr, 0.0) - fmin(wl, 0.0)) * A.cand.rde[k];
    };
    double lam = 0.0, q;
    if (A.cand.n >= 2) {
        lam = fmax(cand_outflow(0), cand_outflow(A.cand.n - 1));        // bins 0 and N_b - 1
        q = __ddiv_rn(__dmul_rn(dtau, lam), A.cfl_e);
        if (!(ceil(q * (1.0 + A.cand.margin)) == ceil(q))) {
            for (int k = 1; k < A.cand.n - 1; ++k) lam = fmax(lam, cand_outflow(k));
            q = __ddiv_rn(__dmul_rn(dtau, lam), A.cfl_e);
        }
    } else {
        for (int i = 0; i < NB; ++i) lam = fmax(lam, lp_outflow(sE, sR, i, a, cr));
        q = __ddiv_rn(__dmul_rn(dtau, lam), A.cfl_e);
    }
    const double need = ceil(q);
    int n = !(need >= 1.0) ? 1 : (need > 2.0e9 ? 2000000000 : (int)need);
    const bool capped = n > A.max_substeps;
    if (capped) n = A.max_substeps;
    const double hdts = 0.5 * __ddiv_rn(dtau, (double)n);      // (dtau / n_sub) / 2, the /2 is exact
    c.a2 = hdts * a;
    c.cr2 = hdts * cr;
    c.ns = n;
    c.cool = fma(c.cr2, sE[0], c.a2) >= 0.0;
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

// Per-lane slice of the bin table: edges E[sub*M .. sub*M+M] and 1/dE of the lane's M bins, held in
// registers (IN_REGS) or re-read from shared memory at each use (large M).  In shared memory the slices
// are stored lane-interleaved (entry i of lane `sub` at [i*32 + sub]): a straight copy of the table would
// put the lanes' slices M*8 bytes apart, i.e. all in the same banks (measured at M = 16: the kernel was
// bound by these 32-way conflicts, l1tex at 94 %).
template <int M, bool IN_REGS, int LANES = 32>
struct LpLaneTab {
    double rE[IN_REGS ? M + 1 : 1], rR[IN_REGS ? M : 1];
    const double *pE, *pR;
    // sE, sR: the plain tables (IN_REGS) or the lane-interleaved ones (lp_fill_interleaved)
    __device__ __forceinline__ void init(const double *sE, const double *sR, int sub)
    {
        if (IN_REGS) {
#pragma unroll
            for (int i = 0; i <= M; ++i) rE[i] = sE[sub * M + i];
#pragma unroll
            for (int i = 0; i < M; ++i) rR[i] = sR[sub * M + i];
            pE = pR = nullptr;
        } else {
            pE = sE + sub;
            pR = sR + sub;
        }
    }
    __device__ __forceinline__ double E(int i) const { return IN_REGS ? rE[i] : pE[i * LANES]; }
    __device__ __forceinline__ double R(int i) const { return IN_REGS ? rR[i] : pR[i * LANES]; }
};

// lane-interleaved copies of the bin table for LpLaneTab<M, false, LANES>: tE[(M+1)*LANES], tR[M*LANES]
// (LANES lanes share a row: 32, or 64 when a pair of warps does)
template <int M, int LANES = 32>
__device__ __forceinline__ void lp_fill_interleaved(const double *tab, int nb, double *tE, double *tR, int tid, int nthreads)
{
    for (int k = tid; k < (M + 1) * LANES; k += nthreads) {
        const int i = k / LANES, lane = k % LANES;
        const int e = lane * M + i;
        tE[k] = e <= nb ? tab[e] : 0.0;
    }
    for (int k = tid; k < M * LANES; k += nthreads) {
        const int i = k / LANES, lane = k % LANES;
        const int b = lane * M + i;
        tR[k] = b < nb ? tab[(nb + 1) + nb + b] : 0.0;
    }
}

// Phase 2 for one row held as M bins per lane over G lanes (32/G rows per warp at once).
// Donor-cell upwind:
//   chi_i <- chi_i - c_i (F_{i+1} - F_i),  F_k = max(w_k,0) chi_{k-1} + min(w_k,0) chi_k,  chi_{-1} = chi_{Nb} = 0,
// with c_i = dts/dE_i.  The coefficients do not change over the substeps, so the update is applied as
// the tridiagonal form it is,
//   chi_i <- D_i chi_i + L_i chi_{i-1} + U_i chi_{i+1},
//   L_i = c_i max(w_i,0),  U_i = -c_i min(w_{i+1},0),  D_i = 1 + c_i (min(w_i,0) - max(w_{i+1},0)),
// three fp64 operations per bin and substep, no selects in the loop.  With W_k = (dts/2) w_k
// = -E_k (a2 + cr2 E_k):  2 max(W,0) = W + |W| and 2 min(W,0) = W - |W| exactly, so
//   L_i = (W_i + |W_i|)/dE_i,  U_i = -(W_{i+1} - |W_{i+1}|)/dE_i,  D_i = 1 + ((W_i - |W_i|) - (W_{i+1} + |W_{i+1}|))/dE_i.
// The zero ghost bins are folded in by L = 0 on the first bin of the row and U = 0 on the last.
// nloop >= c.ns is the trip count shared by the rows a warp works on at once.
template <int M, int G, bool DIAG>
struct LpRow {
    double chi[M], D[M], L[M], U[M];
    double w_first, w_last, s0, s1;
    int ns;

    // first / last: this lane holds the first / the last bin of the row
    template <class Tab>
    __device__ __forceinline__ void setup(const Tab &tab, double a2, double cr2, int ns_, bool first, bool last)
    {
        ns = ns_;
        const double e0 = tab.E(0);
        double w = -e0 * fma(cr2, e0, a2);
        w_first = w;
        double p2 = w + fabs(w), n2 = w - fabs(w);
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const double e = tab.E(i + 1);
            const double w1 = -e * fma(cr2, e, a2);
            const double p2n = w1 + fabs(w1), n2n = w1 - fabs(w1);
            const double r = tab.R(i);
            L[i] = r * p2;
            U[i] = -r * n2n;
            D[i] = fma(r, n2 - p2n, 1.0);
            p2 = p2n;
            n2 = n2n;
            w = w1;
        }
        w_last = w;
        if (first) L[0] = 0.0;
        if (last) U[M - 1] = 0.0;
        s0 = 0.0;
        s1 = 0.0;
    }
    // Rows with a + c_r E_0 >= 0 ("cooling": every edge velocity w_k <= 0) have L = 0 identically, so they
    // need neither L nor the value from the lower neighbour: U_i = -2 W_{i+1}/dE_i, D_i = 1 + 2 W_i/dE_i and
    // chi_i <- D_i chi_i + U_i chi_{i+1}.  These are the same bits the general form gives for such a row
    // (there W + |W| = 0 exactly and the L term adds a zero).
    template <class Tab>
    __device__ __forceinline__ void setup_cool(const Tab &tab, double a2, double cr2, int ns_, bool last)
    {
        ns = ns_;
        const double e0 = tab.E(0);
        double w = -e0 * fma(cr2, e0, a2);
        w_first = w;
        double n2 = w - fabs(w);
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const double e = tab.E(i + 1);
            const double w1 = -e * fma(cr2, e, a2);
            const double n2n = w1 - fabs(w1);
            const double r = tab.R(i);
            U[i] = -r * n2n;
            D[i] = fma(r, n2, 1.0);
            n2 = n2n;
            w = w1;
        }
        w_last = w;
        if (last) U[M - 1] = 0.0;
        s0 = 0.0;
        s1 = 0.0;
    }
    __device__ __forceinline__ void advance_cool()
    {
        const double right = __shfl_down_sync(kFull, chi[0], 1, G);
        if (DIAG) { s0 += chi[0]; s1 += chi[M - 1]; }
        double nx[M];
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const double hi = i == M - 1 ? right : chi[i + 1];
            nx[i] = fma(U[i], hi, D[i] * chi[i]);
        }
#pragma unroll
        for (int i = 0; i < M; ++i) chi[i] = nx[i];
    }
    __device__ __forceinline__ void step_cool(int s)
    {
        constexpr bool kUniform = (G == 32);
        if (kUniform) {
            if (s < ns) advance_cool();
        } else {
            const double right = __shfl_down_sync(kFull, chi[0], 1, G);
            if (s < ns) {
                if (DIAG) { s0 += chi[0]; s1 += chi[M - 1]; }
                double nx[M];
#pragma unroll
                for (int i = 0; i < M; ++i) {
                    const double hi = i == M - 1 ? right : chi[i + 1];
                    nx[i] = fma(U[i], hi, D[i] * chi[i]);
                }
#pragma unroll
                for (int i = 0; i < M; ++i) chi[i] = nx[i];
            }
        }
    }
    // one substep, no test of ns (every lane of the warp calls)
    __device__ __forceinline__ void advance()
    {
        const double left = __shfl_up_sync(kFull, chi[M - 1], 1, G);
        const double right = __shfl_down_sync(kFull, chi[0], 1, G);
        if (DIAG) { s0 += chi[0]; s1 += chi[M - 1]; }
        double nx[M];
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const double lo = i == 0 ? left : chi[i - 1];
            const double hi = i == M - 1 ? right : chi[i + 1];
            nx[i] = fma(U[i], hi, fma(L[i], lo, D[i] * chi[i]));
        }
#pragma unroll
        for (int i = 0; i < M; ++i) chi[i] = nx[i];
    }
    // substep number s (the row takes part while s < ns)
    __device__ __forceinline__ void step(int s)
    {
        constexpr bool kUniform = (G == 32);        // one row per warp: ns is the same on every lane
        if (kUniform) {
            if (s < ns) advance();
        } else {
            const double left = __shfl_up_sync(kFull, chi[M - 1], 1, G);
            const double right = __shfl_down_sync(kFull, chi[0], 1, G);
            if (s < ns) {
                if (DIAG) { s0 += chi[0]; s1 += chi[M - 1]; }
                double nx[M];
#pragma unroll
                for (int i = 0; i < M; ++i) {
                    const double lo = i == 0 ? left : chi[i - 1];
                    const double hi = i == M - 1 ? right : chi[i + 1];
                    nx[i] = fma(U[i], hi, fma(L[i], lo, D[i] * chi[i]));
                }
#pragma unroll
                for (int i = 0; i < M; ++i) chi[i] = nx[i];
            }
        }
    }
    // lost = dts (max(w_Nb,0) sum chi_{Nb-1} - min(w_0,0) sum chi_0),  dts w = 2 W   (all lanes call)
    __device__ __forceinline__ double lost(int sub) const
    {
        double t1 = (sub == G - 1) ? (w_last + fabs(w_last)) * s1 : 0.0;
        double t0 = (sub == 0) ? (w_first - fabs(w_first)) * s0 : 0.0;
        t1 = __shfl_sync(kFull, t1, G - 1, G);
        t0 = __shfl_sync(kFull, t0, 0, G);
        return t1 - t0;
    }
};

// RI independent rows advance together, so that their dependent fp64 chains and shuffles interleave
// (a single row is a chain of ~60 cycles per substep).  nmax = largest n_sub among them (warp-wide).
template <bool COOL, int RI, int M, int G, bool DIAG>
__device__ __forceinline__ void lp_rows_substeps(LpRow<M, G, DIAG> (&row)[RI], int nmin, int nmax)
{
    // the first nmin substeps are common to every row (nmin = smallest n_sub, warp-wide): straight-line
    // code over the RI rows, which the scheduler interleaves
#pragma unroll 1
    for (int s = 0; s < nmin; ++s) {
#pragma unroll
        for (int r = 0; r < RI; ++r) {
            if (COOL) row[r].advance_cool();
            else row[r].advance();
        }
    }
#pragma unroll 1
    for (int s = nmin; s < nmax; ++s) {
#pragma unroll
        for (int r = 0; r < RI; ++r) {
            if (COOL) row[r].step_cool(s);
            else row[r].step(s);
        }
    }
}

// Per-particle phase for one chunk of 32 particles: coefficients into the warp's shared arrays.
template <int NB, bool FUSED>
__device__ __forceinline__ void lp_chunk_phase1(const LpSpectralArgs &A, long long base, int lane,
                                                double px, double py, double pz,
                                                const double *sE, const double *sR, double2 *sAC, int *sNS)
{
    const long long p = base + lane;
    LpCoef c;
    c.a2 = 0.0; c.cr2 = 0.0; c.ns = 0; c.cool = 1;
    if (p < A.np) {
        int nss;
#ifdef LP_DEBUG_SKIP_PHASE1
        c.a2 = 1.0e-3; c.cr2 = 1.0e-12; c.ns = 2; c.cool = 0; nss = 2;
#else
        lp_phase1<NB, FUSED>(A, p, px, py, pz, sE, sR, c, nss);
#endif
        __stcs(A.nsub_ws + p, nss);
        if (A.nsub_user) __stcs(A.nsub_user + p, nss);
    }
    sAC[lane] = make_double2(c.a2, c.cr2);
    sNS[lane] = c.cool ? -c.ns : c.ns;          // the sign carries the cooling flag to the row warps
    __syncwarp();
}

// max of n over the 32/G row groups of a warp (lanes with equal lane % G)
template <int G>
__device__ __forceinline__ int lp_group_max(int n)
{
#pragma unroll
    for (int o = G; o < 32; o <<= 1) n = max(n, __shfl_xor_sync(kFull, n, o));
    return n;
}

// ------------------------------------------------------------------ direct mover (N_b = 512)

constexpr int kDirectThreads = 128;
constexpr int kDirectWarps = kDirectThreads / 32;

// MODE: 0 staged (lp_spectral_update), 1 fused step, 2 fused step that re-sorts (reads through A.perm)
template <int NB, bool DIAG, int MODE>
__global__ void __launch_bounds__(kDirectThreads, 3) lp_spectral_direct_kernel(LpSpectralArgs A)
{
    constexpr bool FUSED = MODE >= 1, PERM = MODE == 2;
    static_assert(NB >= 32, "one row per warp");
    constexpr int G = 32;                     // lanes that share one row
    constexpr int M = NB / G;                 // bins per lane (contiguous)
    constexpr int U = (M <= 2) ? 4 : (M == 4 ? 2 : 1);   // rows in flight per warp

    constexpr bool kTabRegs = (M <= 4);
    // plain copies of the table: the lanes' register slices (M <= 4) are cut from them; with M >= 8 only the
    // per-particle phase would read them (E_0, and every bin when the table has no CFL candidates), and it
    // takes them from global memory instead -- the two row buffers need the shared memory
    __shared__ __align__(16) double sEs[kTabRegs ? NB + 2 : 2];
    __shared__ __align__(16) double sRs[kTabRegs ? NB : 2];
    __shared__ double2 sAC[kDirectWarps][32];
    __shared__ int sNS[kDirectWarps][32];
    const double *sE = kTabRegs ? sEs : A.tab;
    const double *sR = kTabRegs ? sRs : A.tab + (NB + 1) + NB;

    if (kTabRegs) {
        for (int i = threadIdx.x; i <= NB; i += kDirectThreads) sEs[i] = A.tab[i];
        for (int i = threadIdx.x; i < NB; i += kDirectThreads) sRs[i] = A.tab[(NB + 1) + NB + i];
        __syncthreads();
    }

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr bool kStaged = (M >= 8);           // rows through the transposing staging buffer
    static_assert(!kStaged || U == 1, "the staged path keeps one row ahead");
    __shared__ __align__(16) unsigned char sStage[kDirectWarps][kStaged ? LpStage<M>::kBytes : 16];
    __shared__ __align__(16) unsigned char sNext[kDirectWarps][kStaged ? LpStage<M>::kBytes : 16];     // the row fetched ahead
    __shared__ double sET[kTabRegs ? 1 : (M + 1) * 32];
    __shared__ double sRT[kTabRegs ? 1 : M * 32];
    if (!kTabRegs) {
        lp_fill_interleaved<M>(A.tab, NB, sET, sRT, threadIdx.x, kDirectThreads);
        __syncthreads();
    }
    LpLaneTab<M, kTabRegs> tab;
    if (kTabRegs) tab.init(sE, sR, lane);
    else tab.init(sET, sRT, lane);

    const long long nchunks = (A.np + 31) >> 5;
    const long long gw = (long long)blockIdx.x * kDirectWarps + warp;
    const long long nw = (long long)gridDim.x * kDirectWarps;

    for (long long chunk = gw; chunk < nchunks; chunk += nw) {
        const long long base = chunk << 5;
        const bool have = base + lane < A.np;
        // source index of this lane's particle (a re-sort folded into the step reads through the permutation)
        const long long src = have ? (PERM ? (long long)A.perm[base + lane] : base + lane) : 0;
        auto src_of = [&](int j) -> long long { return __shfl_sync(kFull, src, j); };
        const double px = have ? A.xin[src] : 0.0, py = have ? A.yin[src] : 0.0, pz = have ? A.zin[src] : 0.0;
        if (PERM && have) A.id_out[base + lane] = A.id_in[src];
        if constexpr (kStaged) {                            // (staged, U == 1) the next row is fetched a row ahead
            if (base < A.np) LpStage<M>::fetch_async(A.chi_in + src_of(0) * NB, sNext[warp], lane);      // flies during phase 1
        }
        lp_chunk_phase1<NB, FUSED>(A, base, lane, px, py, pz, sE, sR, sAC[warp], sNS[warp]);
        for (int j0 = 0; j0 < 32; j0 += U) {
            double buf[U][M];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const long long pj = base + j0 + u;
                const long long sj = src_of(j0 + u), sj1 = src_of((j0 + u + 1) & 31);      // (all lanes shuffle)
                if (pj < A.np) {
                    if constexpr (kStaged) {
                        LpStage<M>::take(sNext[warp], lane, buf[u]);
                        if (j0 + 1 < 32 && pj + 1 < A.np) LpStage<M>::fetch_async(A.chi_in + sj1 * NB, sNext[warp], lane);
                    } else {
                        lp_load_row<M>(A.chi_in + sj * NB + lane * M, buf[u]);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < M; ++i) buf[u][i] = 0.0;
                }
            }
            LpRow<M, G, DIAG> row[U];
            double2 ac[U];
            int nsr[U];
            int nmax = 0, nmin = 0x7fffffff;
            bool cool = true;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int r = j0 + u;
                ac[u] = sAC[warp][r];
                const int nsv = sNS[warp][r];              // (warp-uniform: every lane reads the same entries)
                cool = cool && nsv <= 0;
                nsr[u] = abs(nsv);
#pragma unroll
                for (int i = 0; i < M; ++i) row[u].chi[i] = buf[u][i];
                nmax = max(nmax, nsr[u]);
                nmin = min(nmin, nsr[u]);
            }
            if (cool) {                                     // every row in flight is a cooling row
#pragma unroll
                for (int u = 0; u < U; ++u) row[u].setup_cool(tab, ac[u].x, ac[u].y, nsr[u], lane == G - 1);
                lp_rows_substeps<true, U, M, G, DIAG>(row, nmin, nmax);
            } else {
#pragma unroll
                for (int u = 0; u < U; ++u) row[u].setup(tab, ac[u].x, ac[u].y, nsr[u], lane == 0, lane == G - 1);
                lp_rows_substeps<false, U, M, G, DIAG>(row, nmin, nmax);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const long long pj = base + j0 + u;
                const double lost = DIAG ? row[u].lost(lane) : 0.0;
                if (pj < A.np) {
                    if constexpr (kStaged) LpStage<M>::store(A.chi_out + pj * NB, sStage[warp], lane, row[u].chi);
                    else lp_store_row<M>(A.chi_out + pj * NB + lane * M, row[u].chi);
                    if (DIAG && lane == 0) {
                        A.lost_ws[pj] = lost;
                        if (A.lost_user) A.lost_user[pj] = lost;
                    }
                }
            }
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------ TMA bulk mover (N_b <= 256)

__device__ __forceinline__ uint32_t lp_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void lp_mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void lp_mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void lp_mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Blocking wait for the phase with the given parity.  try_wait suspends the thread in hardware for
// up to the hinted time, so a waiting warp does not take issue slots from the working ones.
#ifndef LP_MBAR_SUSPEND_NS
#define LP_MBAR_SUSPEND_NS 2000
#endif
__device__ __forceinline__ void lp_mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(bar), "r"(parity), "r"((uint32_t)LP_MBAR_SUSPEND_NS) : "memory");
    } while (!done);
}
// L2 eviction policy for the row stream: rows are touched once per step, the grid records many times
__device__ __forceinline__ uint64_t lp_policy_evict_first()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// global -> shared, completion counted in bytes on an mbarrier (TMA engine, UBLKCP in SASS)
template <bool HINT>
__device__ __forceinline__ void lp_bulk_load(uint32_t dst_smem, const void *src, uint32_t bytes, uint32_t bar,
                                             uint64_t pol)
{
    if (HINT)
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                     ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
    else
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// shared -> global, tracked by bulk async-groups
template <bool HINT>
__device__ __forceinline__ void lp_bulk_store(void *dst, uint32_t src_smem, uint32_t bytes, uint64_t pol)
{
    if (HINT)
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
                     ::"l"(dst), "r"(src_smem), "r"(bytes), "l"(pol) : "memory");
    else
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src_smem), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
template <int N> __device__ __forceinline__ void lp_bulk_wait_read()
{
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void lp_bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void lp_fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Tunables of the bulk mover (overridable at compile time for sweeps; defaults = measured best).
// LP_DEBUG_SKIP_PHASE1 / LP_DEBUG_SKIP_ROWS (never defined in the product build) time one kind of warp alone:
// the first replaces the per-particle phase by constants (results are then meaningless), the second skips
// the row stream.  profiles/r01_spectral_full.md quotes the timings they gave.
#ifndef LP_BULK_MINB
#define LP_BULK_MINB 1          // resident blocks per SM the register allocation is bounded for
#endif
#ifndef LP_BULK_SLOT_SMALL
#define LP_BULK_SLOT_SMALL 4096 // ring slot bytes for N_b <= 64
#endif
#ifndef LP_BULK_MAX_NB
#define LP_BULK_MAX_NB 256      // largest bin count the bulk kernel takes (above: direct kernel)
#endif
#ifndef LP_BULK_SLOT_LARGE
#define LP_BULK_SLOT_LARGE 4096 // ring slot bytes for N_b = 128
#endif
#ifndef LP_BULK_SLOT_HUGE
#define LP_BULK_SLOT_HUGE 4096  // ring slot bytes for N_b >= 256
#endif
#ifndef LP_BULK_DEPTH
#define LP_BULK_DEPTH 3         // ring slots per row warp
#endif
#ifndef LP_BULK_WARPS
#define LP_BULK_WARPS 16        // warps per block (one block per SM)
#endif
// particle warps per block by bin count (the rest are row warps): the per-particle phase costs the same at every
// N_b, the row phase grows with N_b.  Swept in round 2 on workloads 3-5 (fraction of the copy bandwidth):
//   16 bins  8 / 10 / 11 / 12 particle warps: 0.664 / 0.708 / 0.712 / 0.707      32 bins  8 / 9 / 10 / 11: 0.754 / 0.760 / 0.766 / 0.760
//   64 bins  workload 4: 4 / 6 / 7 / 8 / 10: 0.677 / 0.838 / 0.859 / 0.836 / 0.706;  workload 5: 0.665 / 0.804 / 0.813 / 0.759 / 0.744
//   128 bins 3 / 4 / 5 / 6: workload 3 0.818 / 0.922 / 0.944 / 0.871, workload 4 at 128 bins 0.804 / 0.877 / 0.861 / 0.809
//   256 bins 3 / 4 / 5 / 6: 0.839 / 0.828 / 0.811 / 0.780
#ifndef LP_BULK_NP16
#define LP_BULK_NP16 10
#endif
#ifndef LP_BULK_NP32
#define LP_BULK_NP32 10
#endif
#ifndef LP_BULK_NP64
#define LP_BULK_NP64 7
#endif
#ifndef LP_BULK_NP256
#define LP_BULK_NP256 3
#endif
#ifndef LP_BULK_NP128
#define LP_BULK_NP128 4
#endif
// the staged kernel (lp_spectral_update: one stencil per particle instead of three) needs fewer of them; same sweep,
// workload-4 size: 64 bins 5 / 6 / 7 / 8: 3.25 / 3.23 / 3.39 / 3.48 ms; 128 bins 2 / 3 / 4 / 5: 6.93 / 5.90 / 6.28 / 6.39 ms;
// workload 5: 16 bins 6 / 8 / 10 / 12: 0.660 / 0.611 / 0.682 / 0.682 ms; 256 bins 2 / 3 / 4: 3.38 / 3.48 / 3.53 ms
#ifndef LP_BULK_NPS16
#define LP_BULK_NPS16 8
#endif
#ifndef LP_BULK_NPS32
#define LP_BULK_NPS32 8
#endif
#ifndef LP_BULK_NPS64
#define LP_BULK_NPS64 6
#endif
#ifndef LP_BULK_NPS128
#define LP_BULK_NPS128 3
#endif
#ifndef LP_BULK_NPS256
#define LP_BULK_NPS256 2
#endif
#ifndef LP_BULK_L2HINT
#define LP_BULK_L2HINT 1        // row loads and stores of N_b <= 128 carry an L2 evict-first policy (rows are touched
                                // once per step, grid records by many particles); measured +2 % (64 bins) to +8 %
                                // (128 bins) at 16.8M particles, -1.5 % at 256 bins, where it stays off
#endif
#ifndef LP_BULK_COEF_DEPTH
#define LP_BULK_COEF_DEPTH 32   // chunks of coefficients in flight between the two kinds of warp
#endif
#ifndef LP_BULK_CARVEOUT
#define LP_BULK_CARVEOUT cudaSharedmemCarveoutDefault
#endif
#ifndef LP_BULK_M
#define LP_BULK_M 4             // bins per lane (at least N_b/32)
#endif
#ifndef LP_BULK_RI
#define LP_BULK_RI 1            // rows a lane group advances together (ILP)
#endif
#ifndef LP_BULK_GROUP
#define LP_BULK_GROUP 1         // consecutive chunks dealt to a block at a time (power of two)
#endif

template <int NB, bool FUSED>
struct LpBulkCfg {
    static constexpr int M = (NB / 32 > LP_BULK_M) ? NB / 32 : LP_BULK_M;   // bins per lane
    static constexpr int G = NB / M;                              // lanes per row
    static constexpr int PPW = 32 / G;                            // rows a warp works on at once
    static constexpr int ROW_BYTES = NB * 8;
    static constexpr int SLOT_BYTES = NB <= 64 ? LP_BULK_SLOT_SMALL : NB <= 128 ? LP_BULK_SLOT_LARGE : LP_BULK_SLOT_HUGE;     // one ring slot
    static constexpr int R = SLOT_BYTES / ROW_BYTES;              // rows per slot
    static constexpr int GPC = 32 / R;                            // slots ("groups") per chunk of 32 rows
    static constexpr int S = LP_BULK_DEPTH;                       // ring depth per row warp
    static constexpr int NP = FUSED ? (NB <= 16 ? LP_BULK_NP16 : NB == 32 ? LP_BULK_NP32 : NB == 64 ? LP_BULK_NP64 : NB == 128 ? LP_BULK_NP128 : LP_BULK_NP256)
                                    : (NB <= 16 ? LP_BULK_NPS16 : NB == 32 ? LP_BULK_NPS32 : NB == 64 ? LP_BULK_NPS64 : NB == 128 ? LP_BULK_NPS128 : LP_BULK_NPS256);
    static constexpr int NR = LP_BULK_WARPS - NP;                 // particle warps, row warps
    static constexpr int D = LP_BULK_COEF_DEPTH;                  // coefficient ring, in chunks
    static constexpr int THREADS = (NP + NR) * 32;
    static constexpr size_t SMEM_RING = (size_t)NR * S * SLOT_BYTES;
    static constexpr size_t SMEM_TAB = ((size_t)(2 * NB + 2) * 8 + 127) / 128 * 128;
    static constexpr size_t SMEM_COEF = (size_t)D * 32 * (sizeof(double2) + sizeof(int)) + (size_t)D * 2 * sizeof(uint32_t);
    static constexpr size_t SMEM_BAR = ((size_t)(NR * S + 2 * D) * 8 + 127) / 128 * 128;
    static constexpr size_t SMEM_TOTAL = SMEM_RING + SMEM_TAB + SMEM_COEF + SMEM_BAR + 128;
    static constexpr int RI_WANT = (LP_BULK_RI * PPW <= R) ? LP_BULK_RI : R / PPW;
    static constexpr int RI = RI_WANT < 1 ? 1 : RI_WANT;          // rows (per lane group) advanced together
    static_assert(NB % M == 0 && G <= 32 && R % (PPW * RI) == 0 && GPC >= 1 && (GPC & (GPC - 1)) == 0 &&
                  D >= 2 && NP >= 1 && NR >= 1, "ring geometry");
};

// Warp-specialised fused kernel.  A block owns the chunks (32 particles each) blockIdx.x + t*gridDim.x,
// t = 0, 1, ...  Two kinds of warp work on them at their own pace:
//  * particle warps (NP per block, one thread per particle): chunk t goes to particle warp t % NP, which
//    runs phase 1 (push stages when FUSED, gathers, coefficients, n_sub) and leaves (a2, cr2, n_sub) in slot
//    t % D of a shared coefficient ring.  Their time is spent waiting on dependent gathers.
//  * row warps (NR per block): chunk t goes to row warp t % NR, which streams the chunk's rows through its
//    private TMA ring (addresses do not depend on phase 1, so loads run ahead freely), waits for the
//    chunk's coefficients, applies the substeps and stores the rows.
// full[slot] / empty[slot] mbarriers (one arrival each) hand the coefficient slots back and forth.
// Row indices are 32-bit inside the kernel (lp_create limits np to 2^32 - 1); only addresses are 64-bit.
template <int NB, bool DIAG, int MODE>
__global__ void __launch_bounds__(LpBulkCfg<NB, (MODE >= 1)>::THREADS, LP_BULK_MINB) lp_spectral_bulk_kernel(LpSpectralArgs A)
{
    constexpr bool FUSED = MODE >= 1, PERM = MODE == 2;
    using C = LpBulkCfg<NB, (MODE >= 1)>;
    constexpr int G = C::G, M = C::M, PPW = C::PPW, R = C::R, GPC = C::GPC, S = C::S, RI = C::RI;
    constexpr int NP = C::NP, NR = C::NR, D = C::D;

    extern __shared__ __align__(128) unsigned char lp_smem_raw[];
    unsigned char *sm = lp_smem_raw;            // (no pointer casts: keeps the shared address space)
    double *sE = reinterpret_cast<double *>(sm + C::SMEM_RING);
    double *sR = sE + (NB + 2);
    double2 *sAC = reinterpret_cast<double2 *>(sm + C::SMEM_RING + C::SMEM_TAB);
    int *sNS = reinterpret_cast<int *>(sAC + D * 32);
    // Which chunk a coefficient slot holds (sTag) and which chunk was last consumed from it (sDone).  An mbarrier
    // wait only knows the parity of a phase: a warp that gets two phases ahead of a slot's barrier would pass the
    // wait on the phase before last.  With 8 + 8 or 4 + 12 warps and 32 slots that cannot happen (a slot's chunks
    // all belong to one particle warp and one row warp); with 7 + 9, 10 + 6, 3 + 13 it can, so every wait is
    // confirmed against the chunk number and repeated if the slot is not there yet.
    // Ordering.  A wait that passed on the right phase is an acquire paired with the other side's releasing arrive.
    // A wait that passed on a stale phase is not, and the confirmation loop may then leave through the tag alone.  So
    // the tag itself carries the ordering: the writer's lane 0 (behind the __syncwarp that orders the other lanes'
    // sAC / sNS accesses before it) fences and then stores the tag; the reader loads the tag and then fences -- the
    // release and acquire patterns of the PTX memory model on a relaxed (volatile) word.  Whoever reads tag == t
    // therefore sees the slot's coefficients of chunk t (sTag), resp. is past the last read of them (sDone).
    volatile uint32_t *sTag = reinterpret_cast<volatile uint32_t *>(sNS + D * 32);
    volatile uint32_t *sDone = sTag + D;
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(sm + C::SMEM_RING + C::SMEM_TAB + C::SMEM_COEF);
    // bars: [NR*S] ring slots | [D] coefficient slot full | [D] coefficient slot empty

    for (int i = threadIdx.x; i <= NB; i += C::THREADS) sE[i] = A.tab[i];
    for (int i = threadIdx.x; i < NB; i += C::THREADS) sR[i] = A.tab[(NB + 1) + NB + i];
    for (int i = threadIdx.x; i < 2 * D; i += C::THREADS) sTag[i] = 0xffffffffu;
    if (threadIdx.x == 0) {
        for (int i = 0; i < NR * S + 2 * D; ++i) lp_mbar_init(lp_smem_u32(bars + i), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        lp_fence_async_smem();
    }
    __syncthreads();

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t full_u32 = lp_smem_u32(bars + NR * S);
    const uint32_t empty_u32 = full_u32 + 8 * D;
    const uint32_t np = (uint32_t)A.np;
    const uint32_t nchunks = (uint32_t)((A.np + 31) >> 5);
    // Chunks are dealt to the blocks in groups of GS consecutive ones (group g goes to block g % gridDim):
    // neighbouring chunks hold particles of neighbouring cells (the set is sorted by cell), so a block that
    // works through a run of them finds the cell records of the row above or below already in its L1.
    constexpr uint32_t GS = LP_BULK_GROUP;
    const uint32_t ngroups_all = (nchunks + GS - 1) / GS;
    const uint32_t ngb = blockIdx.x < ngroups_all ? (ngroups_all - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    // this block's chunks, t = 0 .. nblk-1 (the last group of all may be short)
    const uint32_t nblk = ngb == 0 ? 0
                          : ngb * GS - (((ngb - 1) * gridDim.x + blockIdx.x == ngroups_all - 1) ? ngroups_all * GS - nchunks : 0);
    auto chunk_start = [&](uint32_t t) -> uint32_t {      // first particle of this block's chunk t
        return ((((t / GS) * gridDim.x + blockIdx.x) * GS) + (t % GS)) << 5;
    };

    if (warp < NP) {
        // ---------------------------------------------------------------- particle warp
        // positions are fetched one chunk ahead, so that their latency is off the dependent chain; when the
        // step re-sorts (A.perm) they are read through the permutation, whose entries are fetched a chunk
        // earlier still, and the ids move with them
        auto chunk_of = [&](uint32_t t) -> uint32_t { return chunk_start(t); };
        const uint32_t *perm = PERM ? A.perm : nullptr;
        auto own_index = [&](uint32_t t, bool &valid) -> uint32_t {      // index of this lane's particle of chunk t
            valid = t < nblk && chunk_of(t) + lane < np;
            return valid ? chunk_of(t) + lane : 0u;
        };
        double nx = 0.0, ny = 0.0, nz = 0.0;
        uint32_t q1 = 0;                    // perm entry of this lane's particle of the chunk after next
        {
            bool v0, v1;
            const uint32_t p0 = own_index(warp, v0), p1 = own_index(warp + NP, v1);
            if (v0) {
                const size_t p = perm ? (size_t)perm[p0] : (size_t)p0;
                nx = __ldcs(A.xin + p); ny = __ldcs(A.yin + p); nz = __ldcs(A.zin + p);   // touched once: streaming
                if (perm) __stcs(A.id_out + p0, __ldcs(A.id_in + p));
            }
            if (perm && v1) q1 = perm[p1];
        }
#pragma unroll 1
        for (uint32_t t = warp; t < nblk; t += NP) {
            const uint32_t cs = t % D, use = t / D;
            const uint32_t base = chunk_of(t);
            const double px = nx, py = ny, pz = nz;
            bool v1, v2;
            const uint32_t p1 = own_index(t + NP, v1), p2 = own_index(t + 2 * NP, v2);
            if (v1) {
                const size_t p = perm ? (size_t)q1 : (size_t)p1;
                nx = __ldcs(A.xin + p); ny = __ldcs(A.yin + p); nz = __ldcs(A.zin + p);   // touched once: streaming
                if (perm) __stcs(A.id_out + p1, __ldcs(A.id_in + p));
            }
            if (perm && v2) q1 = perm[p2];
            if (use >= 1) {                 // the slot's previous chunk (t - D) has been consumed
                lp_mbar_wait(empty_u32 + 8 * cs, (use - 1) & 1u);
                while (sDone[cs] != t - D) { __nanosleep(64); lp_mbar_wait(empty_u32 + 8 * cs, (use - 1) & 1u); }
                __threadfence_block();      // acquire side of sDone
            }
            lp_chunk_phase1<NB, FUSED>(A, (long long)base, lane, px, py, pz, sE, sR, sAC + cs * 32, sNS + cs * 32);
            if (lane == 0) {                // (lp_chunk_phase1 ends with __syncwarp)
                __threadfence_block();      // release side of sTag
                sTag[cs] = t;
                lp_mbar_arrive(full_u32 + 8 * cs);
            }
        }
        return;
    }

    // -------------------------------------------------------------------- row warp
    const int rw = warp - NP;
    const int sub = lane % G, grp = lane / G;
    unsigned char *my_ring = sm + (size_t)rw * S * C::SLOT_BYTES;
    const uint32_t ring_u32 = lp_smem_u32(my_ring);
    const uint32_t bar_u32 = lp_smem_u32(bars + rw * S);
    LpLaneTab<M, true> tab;             // (from shared memory it measured 13 % slower)
    tab.init(sE, sR, sub);

    // this warp's chunks: t = rw, rw + NR, ... (nmy of them); its ring slots ("groups") are numbered
    // j = 0 .. ngroups-1, group j = rows [R * (j % GPC), +R) of its chunk number j / GPC
    const uint32_t nmy = (uint32_t)rw < nblk ? (nblk - rw + NR - 1) / NR : 0;
    const uint32_t ngroups = nmy * GPC;

    constexpr bool kHint = (LP_BULK_L2HINT != 0) && NB <= 128;
    const uint64_t pol = lp_policy_evict_first();
    auto chunk_base = [&](uint32_t k) -> uint32_t { return chunk_start(rw + k * NR); };
    auto group_row0 = [&](uint32_t j) -> uint32_t { return chunk_base(j / GPC) + (j % GPC) * R; };
    auto issue_load = [&](uint32_t j, int slot) {        // lane 0 only: the group's rows are contiguous
        const uint32_t row0 = group_row0(j);
        if (row0 < np) {
            const uint32_t left = np - row0;
            const uint32_t bytes = (left < (uint32_t)R ? left : (uint32_t)R) * C::ROW_BYTES;
            lp_mbar_expect_tx(bar_u32 + 8 * slot, bytes);
            lp_bulk_load<kHint>(ring_u32 + slot * C::SLOT_BYTES, A.chi_in + (size_t)row0 * NB, bytes, bar_u32 + 8 * slot, pol);
        }
    };
    // Re-sort folded into the step: row r of the group comes from row perm[row0 + r] of chi_in -- one bulk copy
    // per row, issued by lane r, all completing on the slot's barrier.  Whole warp calls; `src` = this lane's
    // perm entry for the group (fetched an iteration ahead, so that its latency is not on the issue path).
    const uint32_t *perm = PERM ? A.perm : nullptr;
    auto perm_entry = [&](uint32_t j) -> uint32_t {      // perm[row0(j) + lane], 0 if there is no such row
        if (j >= ngroups || lane >= R) return 0u;
        const uint32_t r = group_row0(j) + lane;
        return r < np ? perm[r] : 0u;
    };
    auto issue_load_perm = [&](uint32_t j, int slot, uint32_t src) {
        const uint32_t row0 = group_row0(j);
        if (row0 < np) {
            const uint32_t left = np - row0;
            const uint32_t nrows = left < (uint32_t)R ? left : (uint32_t)R;
            if (lane == 0) lp_mbar_expect_tx(bar_u32 + 8 * slot, nrows * C::ROW_BYTES);
            __syncwarp();
            if ((uint32_t)lane < nrows)
                lp_bulk_load<kHint>(ring_u32 + slot * C::SLOT_BYTES + lane * C::ROW_BYTES, A.chi_in + (size_t)src * NB,
                                    C::ROW_BYTES, bar_u32 + 8 * slot, pol);
        }
    };
    uint32_t src_next = 0;          // (perm) this lane's entry for the next group to be loaded
    if (perm) {
#pragma unroll
        for (int k = 0; k < S; ++k)
            if ((uint32_t)k < ngroups) issue_load_perm(k, k, perm_entry(k));
        src_next = perm_entry(S);
    } else if (lane == 0) {
#pragma unroll
        for (int k = 0; k < S; ++k)
            if ((uint32_t)k < ngroups) issue_load(k, k);
    }

    uint32_t q = 0;                 // group being consumed
    int slot = 0, pslot = 0;
    uint32_t parity = 0;
#pragma unroll 1
    for (uint32_t k = 0; k < nmy; ++k) {
        const uint32_t t = rw + k * NR;
        const uint32_t cs = t % D, use = t / D;
        const uint32_t base = chunk_base(k);
        const int nchunk = (int)(np - base < 32u ? np - base : 32u);      // rows of this chunk
        lp_mbar_wait(full_u32 + 8 * cs, use & 1u);                         // the chunk's coefficients
        while (sTag[cs] != t) { __nanosleep(64); lp_mbar_wait(full_u32 + 8 * cs, use & 1u); }
        __threadfence_block();              // acquire side of sTag
        const double2 *my_ac = sAC + cs * 32;
        const int *my_ns = sNS + cs * 32;
#pragma unroll 1
        for (int gi = 0; gi < GPC; ++gi, ++q) {
            const int nrows = min(nchunk - gi * R, R);                    // rows of this group (<= 0: none)
#ifndef LP_DEBUG_SKIP_ROWS
            if (nrows > 0) {
                lp_mbar_wait(bar_u32 + 8 * slot, parity);
                double *srow = reinterpret_cast<double *>(my_ring + (size_t)slot * C::SLOT_BYTES);
#pragma unroll 1
                for (int j = 0; j < R; j += PPW * RI) {
                    LpRow<M, G, DIAG> row[RI];
                    double2 ac[RI];
                    int nsr[RI];
                    int nmax = 0, nmin = 0x7fffffff;
                    bool cool = true;
#pragma unroll
                    for (int r = 0; r < RI; ++r) {
                        const int rg = j + r * PPW + grp;           // row within the slot
                        const bool valid = rg < nrows;
                        ac[r] = my_ac[gi * R + rg];
                        const int nsv = valid ? my_ns[gi * R + rg] : 0;
                        cool = cool && nsv <= 0;
                        nsr[r] = abs(nsv);
                        const double *rp = srow + rg * NB + sub * M;
                        if (valid) lp_load_row<M>(rp, row[r].chi);
                        else {
#pragma unroll
                            for (int i = 0; i < M; ++i) row[r].chi[i] = 0.0;
                        }
                        nmax = max(nmax, nsr[r]);
                        nmin = min(nmin, nsr[r]);
                    }
                    nmax = lp_group_max<G>(nmax);
                    nmin = -lp_group_max<G>(-nmin);
                    if (__all_sync(kFull, cool)) {                  // every row in flight is a cooling row
#pragma unroll
                        for (int r = 0; r < RI; ++r) row[r].setup_cool(tab, ac[r].x, ac[r].y, nsr[r], sub == G - 1);
                        lp_rows_substeps<true, RI, M, G, DIAG>(row, nmin, nmax);
                    } else {
#pragma unroll
                        for (int r = 0; r < RI; ++r) row[r].setup(tab, ac[r].x, ac[r].y, nsr[r], sub == 0, sub == G - 1);
                        lp_rows_substeps<false, RI, M, G, DIAG>(row, nmin, nmax);
                    }
#pragma unroll
                    for (int r = 0; r < RI; ++r) {
                        const int rg = j + r * PPW + grp;
                        const double lost = DIAG ? row[r].lost(sub) : 0.0;
                        if (rg < nrows) {
                            lp_store_row<M>(srow + rg * NB + sub * M, row[r].chi);
                            if (DIAG && sub == 0) {
                                const size_t pj = (size_t)base + gi * R + rg;
                                A.lost_ws[pj] = lost;
                                if (A.lost_user) A.lost_user[pj] = lost;
                            }
                        }
                    }
                }
                lp_fence_async_smem();          // generic-proxy writes -> visible to the TMA store
                __syncwarp();
                if (lane == 0)
                    lp_bulk_store<kHint>(A.chi_out + ((size_t)base + gi * R) * NB, ring_u32 + slot * C::SLOT_BYTES,
                                  (uint32_t)nrows * C::ROW_BYTES, pol);
            }
            // refill the slot drained in the previous iteration (its store may still be reading: wait
            // for all but the newest store group), keeping S-1 loads in flight
            if (q >= 1 && q + (S - 1) < ngroups) {
                if (lane == 0) lp_bulk_wait_read<1>();
                if (perm) {
                    __syncwarp();                                   // lane 0's stores have left the slot
                    issue_load_perm(q + (S - 1), pslot, src_next);
                    src_next = perm_entry(q + S);
                } else if (lane == 0) {
                    issue_load(q + (S - 1), pslot);
                }
            }
#endif
            pslot = slot;
            if (++slot == S) { slot = 0; parity ^= 1u; }
        }
        __syncwarp();                                                     // every lane is done with the slot
        if (lane == 0) {
            __threadfence_block();          // release side of sDone
            sDone[cs] = t;
            lp_mbar_arrive(empty_u32 + 8 * cs);
        }
    }
    if (lane == 0) lp_bulk_wait_all();
}

// ------------------------------------------------------------------ launch

template <class K> int lp_blocks_per_sm(K kernel, int threads, size_t smem)
{
    int per_sm = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem);
    return per_sm < 1 ? 1 : per_sm;
}

// blocks_cache: the context's slot for this variant (0 = not set up yet).  Function attributes are per
// device and a context lives on one device, so the set-up runs once per context and variant; a context
// is used by one host thread at a time (lp.h), and cudaFuncSetAttribute itself is thread-safe.
template <int NB, bool DIAG, int MODE>
int launch_variant(const LpSpectralArgs &a, int sm_count, int *blocks_cache, cudaStream_t s)
{
    const long long nchunks = (a.np + 31) >> 5;
    if constexpr (NB <= LP_BULK_MAX_NB) {
        using C = LpBulkCfg<NB, (MODE >= 1)>;
        auto kernel = lp_spectral_bulk_kernel<NB, DIAG, MODE>;
        if (*blocks_cache == 0) {
            if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_TOTAL) != cudaSuccess) return -1;
            if (cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, LP_BULK_CARVEOUT) != cudaSuccess) return -1;
            *blocks_cache = lp_blocks_per_sm(kernel, C::THREADS, C::SMEM_TOTAL);
        }
        const long long want = nchunks;                      // a block takes whole chunks
        const long long cap = (long long)sm_count * *blocks_cache;
        int blocks = (int)(want < cap ? want : cap);
        if (blocks < 1) blocks = 1;
        kernel<<<blocks, C::THREADS, C::SMEM_TOTAL, s>>>(a);
    } else {
        auto kernel = lp_spectral_direct_kernel<NB, DIAG, MODE>;
        if (*blocks_cache == 0) *blocks_cache = lp_blocks_per_sm(kernel, kDirectThreads, 0);
        const long long want = (nchunks + kDirectWarps - 1) / kDirectWarps;
        const long long cap = (long long)sm_count * *blocks_cache;
        int blocks = (int)(want < cap ? want : cap);
        if (blocks < 1) blocks = 1;
        kernel<<<blocks, kDirectThreads, 0, s>>>(a);
    }
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

template <int NB>
int launch_nb(const LpSpectralArgs &a, bool diag, bool fused, int sm_count, int *blocks_cache, cudaStream_t s)
{
    const int mode = fused ? (a.perm ? 2 : 1) : 0;
    int *slot = blocks_cache + (diag ? 3 : 0) + mode;
    if (diag) return mode == 2 ? launch_variant<NB, true, 2>(a, sm_count, slot, s)
                   : mode == 1 ? launch_variant<NB, true, 1>(a, sm_count, slot, s) : launch_variant<NB, true, 0>(a, sm_count, slot, s);
    return mode == 2 ? launch_variant<NB, false, 2>(a, sm_count, slot, s)
         : mode == 1 ? launch_variant<NB, false, 1>(a, sm_count, slot, s) : launch_variant<NB, false, 0>(a, sm_count, slot, s);
}

}  // namespace

int lp_launch_spectral(const LpSpectralArgs &a, int nbins, bool diag, bool fused, int sm_count, int *blocks_cache,
                       cudaStream_t s)
{
    switch (nbins) {
    case 16:  return launch_nb<16>(a, diag, fused, sm_count, blocks_cache, s);
    case 32:  return launch_nb<32>(a, diag, fused, sm_count, blocks_cache, s);
    case 64:  return launch_nb<64>(a, diag, fused, sm_count, blocks_cache, s);
    case 128: return launch_nb<128>(a, diag, fused, sm_count, blocks_cache, s);
    case 256: return launch_nb<256>(a, diag, fused, sm_count, blocks_cache, s);
    case 512: return launch_nb<512>(a, diag, fused, sm_count, blocks_cache, s);
    default:  return -1;
    }
}
