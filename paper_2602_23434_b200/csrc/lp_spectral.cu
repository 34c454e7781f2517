// lp_spectral.cu -- spectral update of every particle (steps a7-a10 of DESIGN.md section 1) and,
// when fused, the two push stages (a5, a6) in front of it.
//
// Phase 1 (one thread = one particle): [push 0, push 1,] gather v, B, rho at x^{n+1}, coefficients,
// CFL substep count.  Phase 2 (one warp = one row, N_b bins spread over the lanes, M = N_b/32
// contiguous bins per lane in registers): n_sub donor-cell upwind substeps of Eq. 6
// with the loss term of Eq. 4; the only cross-lane traffic per substep is one
// shuffle up and one shuffle down of a double.
//
// Two row movers:
//  * lp_spectral_bulk_kernel (N_b <= 128): every warp streams its rows through a private ring of
//    shared-memory slots filled and drained by the TMA engine (cp.async.bulk + mbarrier), so that
//    several KB per warp are in flight while the warp computes, independent of registers.
//  * lp_spectral_direct_kernel (N_b >= 256): rows go global -> registers -> global; these bin counts
//    are bound by the fp64 pipe (n_sub ~ 5-10), not by HBM.
// sm_100a.
#include "lp_device.cuh"

namespace {

constexpr unsigned kFull = 0xffffffffu;

struct __align__(16) LpCoef {      // per-particle scalars handed from phase 1 to phase 2
    double a;      // (1/3) div_mu u^mu
    double cr;     // c_r
    double dts;    // dtau / n_sub
    int ns;        // n_sub (0 = no particle)
    int pad;
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
__device__ __forceinline__ void lp_phase1(const LpSpectralArgs &A, long long p, const double *sE,
                                          const double *sR, LpCoef &c, int &ns_signed)
{
    LpStencil st;
    double px = A.x[p], py = A.y[p], pz = A.z[p];
    double rho_old;
    double qa[4], qb[3];
    if (FUSED) {
        lp_stencil(A.g, px, py, pz, st);
        lp_gather_A(A.cells, st, qa);                       // k1 = v(x^n), rho_old = rho(x^n)
        rho_old = qa[3];
        lp_stencil(A.g, __dadd_rn(px, __dmul_rn(A.dt, qa[0])), __dadd_rn(py, __dmul_rn(A.dt, qa[1])),
                   __dadd_rn(pz, __dmul_rn(A.dt, qa[2])), st);
        double k2[3];
        lp_gather_v(A.cells, st, k2);
        const double hdt = __dmul_rn(0.5, A.dt);
        double pos[3] = { px, py, pz };
        int stt = 0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double xn = __dadd_rn(pos[d], __dmul_rn(hdt, __dadd_rn(qa[d], k2[d])));
            if (A.g.per[d]) xn = lp_wrap_pos(xn, A.g.xlo[d], A.g.xhi[d], A.g.len[d]);
            else if (xn < A.g.xlo[d] || xn >= A.g.xhi[d]) stt |= (1 << d);
            pos[d] = xn;
        }
        px = pos[0]; py = pos[1]; pz = pos[2];
        A.x[p] = px; A.y[p] = py; A.z[p] = pz;
        A.status[p] = stt;
    } else {
        rho_old = A.rho_old[p];
    }
    lp_stencil(A.g, px, py, pz, st);
    lp_gather_A(A.cells, st, qa);
    lp_gather_B(A.cells, st, qb);
    // gamma_g, dtau, c_r (Eq. 4), a (continuity)
    const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(qa[0], qa[0]), __dmul_rn(qa[1], qa[1])), __dmul_rn(qa[2], qa[2]));
    const double b2 = __dadd_rn(__dadd_rn(__dmul_rn(qb[0], qb[0]), __dmul_rn(qb[1], qb[1])), __dmul_rn(qb[2], qb[2]));
    const double gam = __ddiv_rn(1.0, __dsqrt_rn(__dsub_rn(1.0, v2)));
    const double dtau = __ddiv_rn(A.dt, gam);
    const double cr = __dmul_rn(A.kappa, __dadd_rn(__dmul_rn(0.5, b2), A.u_rad));
    const double a = __ddiv_rn(-log(__ddiv_rn(qa[3], rho_old)), __dmul_rn(3.0, dtau));

    // lambda = max_i outflow_i: over the hull-vertex bins (see LpLamCand), or over all bins
    double lam = 0.0;
    if (A.cand.n >= 0) {
        for (int k = 0; k < A.cand.n; ++k) lam = fmax(lam, lp_outflow(sE, sR, A.cand.bin[k], a, cr));
    } else {
        for (int i = 0; i < NB; ++i) lam = fmax(lam, lp_outflow(sE, sR, i, a, cr));
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

// Per-lane slice of the bin table: edges E[sub*M .. sub*M+M] and 1/dE of the lane's M bins, held in
// registers (IN_REGS) or re-read from shared memory at each use (large M).
template <int M, bool IN_REGS>
struct LpLaneTab {
    double rE[IN_REGS ? M + 1 : 1], rR[IN_REGS ? M : 1];
    const double *pE, *pR;
    __device__ __forceinline__ void init(const double *sE, const double *sR, int sub)
    {
        pE = sE + sub * M;
        pR = sR + sub * M;
        if (IN_REGS) {
#pragma unroll
            for (int i = 0; i <= M; ++i) rE[i] = pE[i];
#pragma unroll
            for (int i = 0; i < M; ++i) rR[i] = pR[i];
        }
    }
    __device__ __forceinline__ double E(int i) const { return IN_REGS ? rE[i] : pE[i]; }
    __device__ __forceinline__ double R(int i) const { return IN_REGS ? rR[i] : pR[i]; }
};

// Phase 2 for one row held as M bins per lane over G lanes.  Donor-cell upwind:
//   chi_i <- chi_i - c_i (F_{i+1} - F_i),  F_k = max(w_k,0) chi_{k-1} + min(w_k,0) chi_k,  chi_{-1} = chi_{Nb} = 0,
// with c_i = dts/dE_i.  The coefficients do not change over the substeps, so the update is applied as
// the tridiagonal form it is,
//   chi_i <- D_i chi_i + L_i chi_{i-1} + U_i chi_{i+1},
//   L_i = c_i max(w_i,0),  U_i = -c_i min(w_{i+1},0),  D_i = 1 + c_i (min(w_i,0) - max(w_{i+1},0)),
// three fp64 operations per bin and substep, no selects in the loop.  The zero ghost bins are folded
// in by L = 0 on the first bin of the row and U = 0 on the last.
template <int M, int G, bool DIAG, class Tab>
__device__ __forceinline__ void lp_row_substeps(double (&chi)[M], const Tab &tab, const LpCoef &c, int nloop,
                                                int sub, double &lost)
{
    double D[M], L[M], U[M];
    double w_first, w_last;
    {
        // 2 max(w,0) = w + |w| and 2 min(w,0) = w - |w| are exact; the factor 1/2 goes into h = c_i/2
        const double e0 = tab.E(0);
        double w = -e0 * fma(c.cr, e0, c.a);
        w_first = w;
        double p2 = w + fabs(w), n2 = w - fabs(w);
        const double hdts = 0.5 * c.dts;
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const double e = tab.E(i + 1);
            const double w1 = -e * fma(c.cr, e, c.a);
            const double p2n = w1 + fabs(w1), n2n = w1 - fabs(w1);
            const double h = hdts * tab.R(i);
            L[i] = h * p2;
            U[i] = -h * n2n;
            D[i] = fma(h, n2 - p2n, 1.0);
            p2 = p2n;
            n2 = n2n;
            w = w1;
        }
        w_last = w;
        if (sub == 0) L[0] = 0.0;
        if (sub == G - 1) U[M - 1] = 0.0;
    }
    double s0 = 0.0, s1 = 0.0;
    constexpr bool kUniform = (G == 32);        // one row per warp: nloop == c.ns for every lane
    for (int s = 0; s < nloop; ++s) {
        const double left = __shfl_up_sync(kFull, chi[M - 1], 1, G);
        const double right = __shfl_down_sync(kFull, chi[0], 1, G);
        if (kUniform || s < c.ns) {
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
    if (DIAG) {
        double t1 = (sub == G - 1) ? fmax(w_last, 0.0) * s1 : 0.0;
        double t0 = (sub == 0) ? fmin(w_first, 0.0) * s0 : 0.0;
        t1 = __shfl_sync(kFull, t1, G - 1, G);
        t0 = __shfl_sync(kFull, t0, 0, G);
        lost = c.dts * (t1 - t0);
    }
}

template <int NB, bool FUSED>
__device__ __forceinline__ void lp_chunk_phase1(const LpSpectralArgs &A, long long base, int lane,
                                                const double *sE, const double *sR, LpCoef *slot)
{
    const long long p = base + lane;
    LpCoef c;
    c.a = 0.0; c.cr = 0.0; c.dts = 0.0; c.ns = 0; c.pad = 0;
    if (p < A.np) {
        int nss;
        lp_phase1<NB, FUSED>(A, p, sE, sR, c, nss);
        A.nsub_ws[p] = nss;
        if (A.nsub_user) A.nsub_user[p] = nss;
    }
    slot[lane] = c;
    __syncwarp();
}

// ------------------------------------------------------------------ direct mover (N_b >= 256)

constexpr int kDirectThreads = 256;
constexpr int kDirectWarps = kDirectThreads / 32;

template <int NB, bool DIAG, bool FUSED>
__global__ void __launch_bounds__(kDirectThreads) lp_spectral_direct_kernel(LpSpectralArgs A)
{
    constexpr int G = NB >= 32 ? 32 : NB;     // lanes that share one row
    constexpr int M = NB / G;                 // bins per lane (contiguous)
    constexpr int PPW = 32 / G;               // rows a warp works on at once
    constexpr int ROWS = 32 / PPW;            // row iterations per chunk of 32 particles
    constexpr int U = (M <= 2) ? 4 : (M == 4 ? 2 : 1);   // rows in flight per warp

    __shared__ __align__(16) double sE[NB + 2];
    __shared__ __align__(16) double sR[NB];
    __shared__ LpCoef sC[kDirectWarps][32];

    for (int i = threadIdx.x; i <= NB; i += kDirectThreads) sE[i] = A.tab[i];
    for (int i = threadIdx.x; i < NB; i += kDirectThreads) sR[i] = A.tab[(NB + 1) + NB + i];
    __syncthreads();

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane % G, grp = lane / G;
    LpLaneTab<M, (M <= 4)> tab;
    tab.init(sE, sR, sub);

    const long long nchunks = (A.np + 31) >> 5;
    const long long gw = (long long)blockIdx.x * kDirectWarps + warp;
    const long long nw = (long long)gridDim.x * kDirectWarps;

    for (long long chunk = gw; chunk < nchunks; chunk += nw) {
        const long long base = chunk << 5;
        lp_chunk_phase1<NB, FUSED>(A, base, lane, sE, sR, sC[warp]);
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
                lp_row_substeps<M, G, DIAG>(buf[u], tab, c, nloop, sub, lost);
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

// ------------------------------------------------------------------ TMA bulk mover (N_b <= 128)

__device__ __forceinline__ uint32_t lp_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void lp_mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void lp_mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void lp_mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}
// global -> shared, completion counted in bytes on an mbarrier (TMA engine, UBLKCP in SASS)
__device__ __forceinline__ void lp_bulk_load(uint32_t dst_smem, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// shared -> global, tracked by bulk async-groups
__device__ __forceinline__ void lp_bulk_store(void *dst, uint32_t src_smem, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src_smem), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
template <int N> __device__ __forceinline__ void lp_bulk_wait_read()
{
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void lp_bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void lp_fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <int NB>
struct LpBulkCfg {
    static constexpr int G = NB >= 32 ? 32 : NB;
    static constexpr int M = NB / G;
    static constexpr int PPW = 32 / G;
    static constexpr int ROW_BYTES = NB * 8;
    static constexpr int SLOT_BYTES = NB <= 64 ? 2048 : 4096;     // one ring slot
    static constexpr int R = SLOT_BYTES / ROW_BYTES;              // rows per slot: 16, 8, 4, 4
    static constexpr int GPC = 32 / R;                            // slots ("groups") per chunk of 32 rows
    static constexpr int S = 3;                                   // ring depth per warp
    static constexpr int WARPS = 4;                               // warps per block
    static constexpr int THREADS = WARPS * 32;
    static constexpr size_t SMEM_RING = (size_t)WARPS * S * SLOT_BYTES;
    static constexpr size_t SMEM_TAB = ((size_t)(2 * NB + 2) * 8 + 127) / 128 * 128;
    static constexpr size_t SMEM_COEF = (size_t)WARPS * 32 * sizeof(LpCoef);
    static constexpr size_t SMEM_BAR = 128;
    static constexpr size_t SMEM_TOTAL = SMEM_RING + SMEM_TAB + SMEM_COEF + SMEM_BAR + 128;
    static_assert(R % PPW == 0 && GPC >= 1 && WARPS * S * 8 <= (int)SMEM_BAR, "ring geometry");
};

template <int NB, bool DIAG, bool FUSED>
__global__ void __launch_bounds__(LpBulkCfg<NB>::THREADS) lp_spectral_bulk_kernel(LpSpectralArgs A)
{
    using C = LpBulkCfg<NB>;
    constexpr int G = C::G, M = C::M, PPW = C::PPW, R = C::R, GPC = C::GPC, S = C::S;

    extern __shared__ __align__(128) unsigned char lp_smem_raw[];
    unsigned char *sm = lp_smem_raw;            // (no pointer casts: keeps the shared address space)
    unsigned char *ring = sm;
    double *sE = reinterpret_cast<double *>(sm + C::SMEM_RING);
    double *sR = sE + (NB + 2);
    LpCoef *sC = reinterpret_cast<LpCoef *>(sm + C::SMEM_RING + C::SMEM_TAB);
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(sm + C::SMEM_RING + C::SMEM_TAB + C::SMEM_COEF);

    for (int i = threadIdx.x; i <= NB; i += C::THREADS) sE[i] = A.tab[i];
    for (int i = threadIdx.x; i < NB; i += C::THREADS) sR[i] = A.tab[(NB + 1) + NB + i];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane % G, grp = lane / G;
    unsigned char *my_ring = ring + (size_t)warp * S * C::SLOT_BYTES;
    const uint32_t ring_u32 = lp_smem_u32(my_ring);
    const uint32_t bar_u32 = lp_smem_u32(bars + warp * S);
    LpCoef *my_coef = sC + warp * 32;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < S; ++s) lp_mbar_init(bar_u32 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        lp_fence_async_smem();
    }
    __syncthreads();

    LpLaneTab<M, true> tab;
    tab.init(sE, sR, sub);

    // this warp's chunks: gw, gw + nw, ...; its slots ("groups") are numbered q = 0 .. ngroups-1
    const long long nchunks = (A.np + 31) >> 5;
    const long long gw = (long long)blockIdx.x * C::WARPS + warp;
    const long long nw = (long long)gridDim.x * C::WARPS;
    const long long nmy = gw < nchunks ? (nchunks - gw + nw - 1) / nw : 0;
    const long long ngroups = nmy * GPC;

    auto rows_at = [&](long long row0) -> int {
        const long long left = A.np - row0;
        return left >= R ? R : (left > 0 ? (int)left : 0);
    };
    // loader state (lane 0): next group to load = (chunk base lbase, group lgi) into slot lslot
    long long lbase = gw << 5, lq = 0;
    int lgi = 0, lslot = 0;
    auto issue_next_load = [&]() {              // lane 0 only; advances the loader state
        if (lq < ngroups) {
            const long long row0 = lbase + (long long)lgi * R;
            const int nrows = rows_at(row0);
            if (nrows > 0) {
                const uint32_t bytes = (uint32_t)nrows * C::ROW_BYTES;
                lp_mbar_expect_tx(bar_u32 + 8 * lslot, bytes);
                lp_bulk_load(ring_u32 + lslot * C::SLOT_BYTES, A.chi_in + row0 * NB, bytes, bar_u32 + 8 * lslot);
            }
            ++lq;
            if (++lgi == GPC) { lgi = 0; lbase += nw << 5; }
            if (++lslot == S) lslot = 0;
        }
    };
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < S; ++k) issue_next_load();
    }

    long long base = gw << 5;
    int gi = 0, slot = 0;
    uint32_t parity = 0;
    for (long long q = 0; q < ngroups; ++q) {
        if (gi == 0)        // a new chunk of 32 particles: per-particle phase while the rows fly in
            lp_chunk_phase1<NB, FUSED>(A, base, lane, sE, sR, my_coef);
        const long long row0 = base + (long long)gi * R;
        const int nrows = rows_at(row0);
        if (nrows > 0) {
            lp_mbar_wait(bar_u32 + 8 * slot, parity);
            double *srow = reinterpret_cast<double *>(my_ring + (size_t)slot * C::SLOT_BYTES);
            const LpCoef *cf = my_coef + gi * R;
#pragma unroll 2
            for (int j = 0; j < R; j += PPW) {
                const int rg = j + grp;                 // row within the slot
                const bool valid = rg < nrows;
                const LpCoef c = cf[rg];
                double chi[M];
                double *rp = srow + rg * NB + sub * M;
                if (valid) lp_load_row<M>(rp, chi);
                else {
#pragma unroll
                    for (int i = 0; i < M; ++i) chi[i] = 0.0;
                }
                int nloop = valid ? c.ns : 0;
                if (PPW > 1) nloop = max(nloop, __shfl_xor_sync(kFull, nloop, 16));
                double lost = 0.0;
                lp_row_substeps<M, G, DIAG>(chi, tab, c, nloop, sub, lost);
                if (valid) {
                    lp_store_row<M>(rp, chi);
                    if (DIAG && sub == 0) {
                        A.lost_ws[row0 + rg] = lost;
                        if (A.lost_user) A.lost_user[row0 + rg] = lost;
                    }
                }
            }
            lp_fence_async_smem();          // generic-proxy writes -> visible to the TMA store
            __syncwarp();
            if (lane == 0)
                lp_bulk_store(A.chi_out + row0 * NB, ring_u32 + slot * C::SLOT_BYTES, (uint32_t)nrows * C::ROW_BYTES);
        }
        // refill the slot drained in the previous iteration (its store may still be reading: wait for
        // all but the newest store group), keeping S-1 loads in flight
        if (q >= 1 && lane == 0 && lq < ngroups) {
            lp_bulk_wait_read<1>();
            issue_next_load();
        }
        __syncwarp();
        if (++gi == GPC) { gi = 0; base += nw << 5; }
        if (++slot == S) { slot = 0; parity ^= 1u; }
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

template <int NB, bool DIAG, bool FUSED>
int launch_variant(const LpSpectralArgs &a, int sm_count, cudaStream_t s)
{
    const long long nchunks = (a.np + 31) >> 5;
    if constexpr (NB <= 128) {
        using C = LpBulkCfg<NB>;
        auto kernel = lp_spectral_bulk_kernel<NB, DIAG, FUSED>;
        static bool configured = false;
        if (!configured) {
            if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_TOTAL) != cudaSuccess) return -1;
            configured = true;
        }
        const long long want = (nchunks + C::WARPS - 1) / C::WARPS;
        const long long cap = (long long)sm_count * lp_blocks_per_sm(kernel, C::THREADS, C::SMEM_TOTAL);
        int blocks = (int)(want < cap ? want : cap);
        if (blocks < 1) blocks = 1;
        kernel<<<blocks, C::THREADS, C::SMEM_TOTAL, s>>>(a);
    } else {
        auto kernel = lp_spectral_direct_kernel<NB, DIAG, FUSED>;
        const long long want = (nchunks + kDirectWarps - 1) / kDirectWarps;
        const long long cap = (long long)sm_count * lp_blocks_per_sm(kernel, kDirectThreads, 0);
        int blocks = (int)(want < cap ? want : cap);
        if (blocks < 1) blocks = 1;
        kernel<<<blocks, kDirectThreads, 0, s>>>(a);
    }
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

template <int NB>
int launch_nb(const LpSpectralArgs &a, bool diag, bool fused, int sm_count, cudaStream_t s)
{
    if (diag) return fused ? launch_variant<NB, true, true>(a, sm_count, s) : launch_variant<NB, true, false>(a, sm_count, s);
    return fused ? launch_variant<NB, false, true>(a, sm_count, s) : launch_variant<NB, false, false>(a, sm_count, s);
}

}  // namespace

int lp_launch_spectral(const LpSpectralArgs &a, int nbins, bool diag, bool fused, int sm_count, cudaStream_t s)
{
    switch (nbins) {
    case 16:  return launch_nb<16>(a, diag, fused, sm_count, s);
    case 32:  return launch_nb<32>(a, diag, fused, sm_count, s);
    case 64:  return launch_nb<64>(a, diag, fused, sm_count, s);
    case 128: return launch_nb<128>(a, diag, fused, sm_count, s);
    case 256: return launch_nb<256>(a, diag, fused, sm_count, s);
    case 512: return launch_nb<512>(a, diag, fused, sm_count, s);
    default:  return -1;
    }
}
