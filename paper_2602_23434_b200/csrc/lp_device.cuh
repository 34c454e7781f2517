// lp_device.cuh -- device helpers of the CUDA path: cell index, trilinear stencil, gather.
//
// Arithmetic contract (reading R14): everything that decides an index or a position
// uses the explicit round-to-nearest intrinsics (__dadd_rn, __dmul_rn, ...), which nvcc never
// contracts into an FMA, in a fixed order.  Each is one correctly rounded IEEE-754 operation, so
// cell keys, sort order and positions are reproducible bit for bit.
#pragma once
#include <cuda_runtime.h>
#include "lp_internal.h"

// floor-mod for an index far outside the grid (kept out of line: the integer division is long)
static __device__ __noinline__ int lp_wrap_far(int i, int n)
{
    int m = i % n;
    return m < 0 ? m + n : m;
}

__device__ __forceinline__ int lp_wrap(int i, int n, int periodic)
{
    if (periodic) {
        if (i >= -n && i < 2 * n) return i < 0 ? i + n : (i >= n ? i - n : i);   // the usual case, no division
        return lp_wrap_far(i, n);
    }
    return min(max(i, 0), n - 1);
}

// containing cell of one coordinate: floor((x - lo) * inv_dx), clamped   (R15)
__device__ __forceinline__ int lp_cell_1d(double x, double lo, double inv_dx, int n)
{
    double s = __dmul_rn(__dsub_rn(x, lo), inv_dx);
    int c = (int)floor(s);
    return min(max(c, 0), n - 1);
}

__device__ __forceinline__ uint32_t lp_cell_key(const LpGeom &g, double x, double y, double z)
{
    int ci = lp_cell_1d(x, g.xlo[0], g.inv_dx[0], g.nx);
    int cj = lp_cell_1d(y, g.xlo[1], g.inv_dx[1], g.ny);
    int ck = lp_cell_1d(z, g.xlo[2], g.inv_dx[2], g.nz);
    return (uint32_t)((ck * g.ny + cj) * g.nx + ci);
}

// Trilinear stencil of a position: 8 cell indices and weights, corners ordered z outer, y, x inner;
// weight = (wz*wy)*wx.  Cell-centred data: s = (x - lo)*inv_dx - 1/2, i0 = floor(s), f = s - i0.
struct LpStencil {
    unsigned int c[8];          // cell index < 2^31 (lp_create rejects larger grids)
    double w[8];
};

__device__ __forceinline__ void lp_axis(double x, double lo, double inv_dx, int n, int periodic,
                                        int &i0, int &i1, double &w0, double &w1)
{
    double s = __dsub_rn(__dmul_rn(__dsub_rn(x, lo), inv_dx), 0.5);
    double fl = floor(s);
    double f = __dsub_rn(s, fl);
    int b = (int)fl;
    i0 = lp_wrap(b, n, periodic);
    if (periodic) i1 = (i0 + 1 == n) ? 0 : i0 + 1;          // floor-mod of b + 1
    else i1 = min(max(b + (b != 0x7fffffff), 0), n - 1);   // (the conversion saturates for positions absurdly far out: no overflow)
    w0 = __dsub_rn(1.0, f);
    w1 = f;
}

__device__ __forceinline__ void lp_stencil(const LpGeom &g, double x, double y, double z, LpStencil &st)
{
    int ii[2], jj[2], kk[2];
    double wx[2], wy[2], wz[2];
    lp_axis(x, g.xlo[0], g.inv_dx[0], g.nx, g.per[0], ii[0], ii[1], wx[0], wx[1]);
    lp_axis(y, g.xlo[1], g.inv_dx[1], g.ny, g.per[1], jj[0], jj[1], wy[0], wy[1]);
    lp_axis(z, g.xlo[2], g.inv_dx[2], g.nz, g.per[2], kk[0], kk[1], wz[0], wz[1]);
#pragma unroll
    for (int cz = 0; cz < 2; ++cz)
#pragma unroll
        for (int cy = 0; cy < 2; ++cy)
#pragma unroll
            for (int cx = 0; cx < 2; ++cx) {
                int n = (cz * 2 + cy) * 2 + cx;
                st.w[n] = __dmul_rn(__dmul_rn(wz[cz], wy[cy]), wx[cx]);
                st.c[n] = (unsigned int)((kk[cz] * g.ny + jj[cy]) * g.nx + ii[cx]);
            }
}

__device__ __forceinline__ double lp_acc(double acc, double w, double q) { return __dadd_rn(acc, __dmul_rn(w, q)); }

// One 32-byte cell record per request: sm_100a has 256-bit global loads (LDG.E.256), which halve
// the L1 request count of the gather (the per-particle phase is bound by L1 requests, one per lane
// and divergent address, not by bytes).
struct LpRec { double a, b, c, d; };
// The load carries an L2 evict-last policy: a cell's record is needed again by the particles of the
// neighbouring rows and planes, long after the row stream (evict-first, lp_spectral.cu) has passed.
__device__ __forceinline__ LpRec lp_ldg_rec(const double4 *p)
{
    LpRec r;
    unsigned long long pol;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    asm("ld.global.nc.L2::cache_hint.v4.f64 {%0,%1,%2,%3}, [%4], %5;"
        : "=d"(r.a), "=d"(r.b), "=d"(r.c), "=d"(r.d) : "l"(p), "l"(pol));
    return r;
}

// The eight (vx, vy, vz, rho) corner records of a stencil, kept in registers across the gathers of
// one step: x^n, x* and x^{n+1} of a particle mostly share their stencil (|v| dt < dx/2), and a
// record that is already in registers costs no L1 request.  The records are reloaded only by the
// lanes whose stencil moved; values are the same bits either way.
struct LpCornersA {
    LpRec r[8];
    unsigned int c0, c7;        // cells of corners 0 and 7 of the loaded stencil (they fix all eight)
    __device__ __forceinline__ void load(const LpCells &cells, const LpStencil &st)
    {
#pragma unroll
        for (int n = 0; n < 8; ++n) r[n] = lp_ldg_rec(cells.recA + (size_t)cells.stride * st.c[n]);
        c0 = st.c[0];
        c7 = st.c[7];
    }
    __device__ __forceinline__ void update(const LpCells &cells, const LpStencil &st)
    {
        if (st.c[0] != c0 || st.c[7] != c7) load(cells, st);
    }
    // (vx, vy, vz, rho)
    __device__ __forceinline__ void gather4(const LpStencil &st, double out[4]) const
    {
        out[0] = out[1] = out[2] = out[3] = 0.0;
#pragma unroll
        for (int n = 0; n < 8; ++n) {
            out[0] = lp_acc(out[0], st.w[n], r[n].a);
            out[1] = lp_acc(out[1], st.w[n], r[n].b);
            out[2] = lp_acc(out[2], st.w[n], r[n].c);
            out[3] = lp_acc(out[3], st.w[n], r[n].d);
        }
    }
    // (vx, vy, vz)
    __device__ __forceinline__ void gather3(const LpStencil &st, double out[3]) const
    {
        out[0] = out[1] = out[2] = 0.0;
#pragma unroll
        for (int n = 0; n < 8; ++n) {
            out[0] = lp_acc(out[0], st.w[n], r[n].a);
            out[1] = lp_acc(out[1], st.w[n], r[n].b);
            out[2] = lp_acc(out[2], st.w[n], r[n].c);
        }
    }
};

// (vx, vy, vz, rho) from record A
__device__ __forceinline__ void lp_gather_A(const LpCells &cells, const LpStencil &st, double out[4])
{
    LpCornersA k;
    k.load(cells, st);
    k.gather4(st, out);
}

// (vx, vy, vz) only: rho is loaded (same 32-byte record) but not accumulated
__device__ __forceinline__ void lp_gather_v(const LpCells &cells, const LpStencil &st, double out[3])
{
    LpCornersA k;
    k.load(cells, st);
    k.gather3(st, out);
}

// (bx, by, bz) from record B, in two halves so that the loads can be issued ahead of other work
struct LpCornersB {
    LpRec r[8];
    __device__ __forceinline__ void load(const LpCells &cells, const LpStencil &st)
    {
#pragma unroll
        for (int n = 0; n < 8; ++n) r[n] = lp_ldg_rec(cells.recB + (size_t)cells.stride * st.c[n]);
    }
    __device__ __forceinline__ void gather3(const LpStencil &st, double out[3]) const
    {
        out[0] = out[1] = out[2] = 0.0;
#pragma unroll
        for (int n = 0; n < 8; ++n) {
            out[0] = lp_acc(out[0], st.w[n], r[n].a);
            out[1] = lp_acc(out[1], st.w[n], r[n].b);
            out[2] = lp_acc(out[2], st.w[n], r[n].c);
        }
    }
};

__device__ __forceinline__ void lp_gather_B(const LpCells &cells, const LpStencil &st, double out[3])
{
    LpCornersB k;
    k.load(cells, st);
    k.gather3(st, out);
}

// periodic wrap into [lo, hi): x -= L*floor((x - lo)/L); a result >= hi becomes lo   (R15)
// For 0 <= x - lo < L (both rounded) the rounded quotient is in [0, 1): its floor is 0 and x is
// unchanged, so the division is skipped there; the result is bit-identical either way.
__device__ __forceinline__ double lp_wrap_pos(double x, double lo, double hi, double L)
{
    const double d = __dsub_rn(x, lo);
    if (!(d >= 0.0 && d < L)) {
        const double t = floor(__ddiv_rn(d, L));
        x = __dsub_rn(x, __dmul_rn(L, t));
    }
    return x >= hi ? lo : x;
}

// The per-particle part every spectral kernel starts with: [FUSED: the two push stages a5, a6 (same arithmetic as
// lp_push0/1_kernel), run on the same thread so that k1, x*, rho_old never leave registers;
// x^{n+1} and the outside-box status are written], then the gathers at x^{n+1} and the coefficients a7:
// dtau = dt/gamma_g, c_r (Eq. 4), a = (1/3) div_mu u^mu through continuity
// (PAPER.md:105).  Not FUSED: (px, py, pz) is x^{n+1} and rho_old comes from push stage 0.
template <bool FUSED>
__device__ __forceinline__ void lp_particle_coefficients(const LpGeom &g, const LpCells &cells, double dt, double kappa,
                                                         double u_rad, double *x, double *y, double *z, int32_t *status,
                                                         const double *rho_old_in, long long p, double px, double py,
                                                         double pz, double &a, double &cr, double &dtau)
{
    LpStencil st;
    LpCornersA ka;
    LpCornersB kb;
    double rho_old;
    double qa[4], qb[3];
    if (FUSED) {
        lp_stencil(g, px, py, pz, st);
        ka.load(cells, st);
        // B is gathered last, at x^{n+1}, whose cells are these or their neighbours.  With split record arrays
        // start the B halves of the four x-lower corners on their way from DRAM to L2 now (every prefetch is an
        // L1 request, and eight cost more than they save); in a 64-byte record the B half arrives in L2 with A.
        if (cells.stride == 1) {
#pragma unroll
            for (int n = 0; n < 8; n += 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(cells.recB + st.c[n]));
        }
        ka.gather4(st, qa);                                 // k1 = v(x^n), rho_old = rho(x^n)
        rho_old = qa[3];
        lp_stencil(g, __dadd_rn(px, __dmul_rn(dt, qa[0])), __dadd_rn(py, __dmul_rn(dt, qa[1])),
                   __dadd_rn(pz, __dmul_rn(dt, qa[2])), st);
        double k2[3];
        ka.update(cells, st);
        ka.gather3(st, k2);
        const double hdt = __dmul_rn(0.5, dt);
        double pos[3] = { px, py, pz };
        int stt = 0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double xn = __dadd_rn(pos[d], __dmul_rn(hdt, __dadd_rn(qa[d], k2[d])));
            if (g.per[d]) xn = lp_wrap_pos(xn, g.xlo[d], g.xhi[d], g.len[d]);
            else if (xn < g.xlo[d] || xn >= g.xhi[d]) stt |= (1 << d);
            pos[d] = xn;
        }
        px = pos[0]; py = pos[1]; pz = pos[2];
        __stcs(x + p, px); __stcs(y + p, py); __stcs(z + p, pz);
        __stcs(status + p, stt);
        lp_stencil(g, px, py, pz, st);
        ka.update(cells, st);
    } else {
        rho_old = rho_old_in[p];
        lp_stencil(g, px, py, pz, st);
        ka.load(cells, st);
    }
    ka.gather4(st, qa);
    kb.load(cells, st);       // (issued after A is consumed: holding both record sets spills registers)
    kb.gather3(st, qb);
    // gamma_g, dtau, c_r (Eq. 4), a (continuity)
    const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(qa[0], qa[0]), __dmul_rn(qa[1], qa[1])), __dmul_rn(qa[2], qa[2]));
    const double b2 = __dadd_rn(__dadd_rn(__dmul_rn(qb[0], qb[0]), __dmul_rn(qb[1], qb[1])), __dmul_rn(qb[2], qb[2]));
    const double gam = __ddiv_rn(1.0, __dsqrt_rn(__dsub_rn(1.0, v2)));
    dtau = __ddiv_rn(dt, gam);
    cr = __dmul_rn(kappa, __dadd_rn(__dmul_rn(0.5, b2), u_rad));
    a = __ddiv_rn(-log(__ddiv_rn(qa[3], rho_old)), __dmul_rn(3.0, dtau));
}

// Row <-> lane slices through a per-warp staging buffer, for M >= 8 bins per lane.  A lane's slice is M*8
// bytes of the row, so loading it directly makes every 16-byte load instruction of the warp touch 32
// different 128-byte lines (measured at M = 16: ~500 L1 wavefronts per row, the kernel's bound after the
// table fix).  Instead the warp moves the row with fully coalesced 16-byte accesses and transposes in shared
// memory; slices are padded by 16 bytes so that both sides are free of bank conflicts.
template <int M>
struct LpStage {
    static constexpr int kSliceBytes = M * 8 + 16;                 // padded slice of one lane
    static constexpr int kBytes = 32 * kSliceBytes;
    // 16-byte unit e of the row (0 .. 2M*... ) lives at:
    static __device__ __forceinline__ int unit_offset(int e) { return (e / (M / 2)) * kSliceBytes + (e % (M / 2)) * 16; }

    // the row's coalesced 16-byte pieces into registers (issued early: a row ahead of its use)
    static __device__ __forceinline__ void fetch(const double *__restrict__ grow, int lane, double2 (&t)[M / 2])
    {
#pragma unroll
        for (int k = 0; k < M / 2; ++k) t[k] = *reinterpret_cast<const double2 *>(grow + 2 * (k * 32 + lane));
    }
    // fetched pieces -> this lane's slice
    static __device__ __forceinline__ void place(const double2 (&t)[M / 2], unsigned char *stage, int lane, double (&v)[M])
    {
#pragma unroll
        for (int k = 0; k < M / 2; ++k) *reinterpret_cast<double2 *>(stage + unit_offset(k * 32 + lane)) = t[k];
        __syncwarp();
#pragma unroll
        for (int j = 0; j < M / 2; ++j) {
            const double2 u = *reinterpret_cast<const double2 *>(stage + lane * kSliceBytes + j * 16);
            v[2 * j] = u.x;
            v[2 * j + 1] = u.y;
        }
        __syncwarp();
    }
    // The same without registers in between: the row's 16-byte pieces go straight from global memory to their
    // place in a stage buffer (cp.async, LDGSTS) and are collected by take() once they have landed -- a row can
    // be fetched a whole row ahead at no register cost.
    static __device__ __forceinline__ void fetch_async(const double *__restrict__ grow, unsigned char *stage, int lane)
    {
#pragma unroll
        for (int k = 0; k < M / 2; ++k) {
            const uint32_t dst = (uint32_t)__cvta_generic_to_shared(stage + unit_offset(k * 32 + lane));
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(grow + 2 * (k * 32 + lane)) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    static __device__ __forceinline__ void take(unsigned char *stage, int lane, double (&v)[M])
    {
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncwarp();
#pragma unroll
        for (int j = 0; j < M / 2; ++j) {
            const double2 u = *reinterpret_cast<const double2 *>(stage + lane * kSliceBytes + j * 16);
            v[2 * j] = u.x;
            v[2 * j + 1] = u.y;
        }
        __syncwarp();
    }
    static __device__ __forceinline__ void store(double *__restrict__ grow, unsigned char *stage, int lane,
                                                 const double (&v)[M])
    {
#pragma unroll
        for (int j = 0; j < M / 2; ++j)
            *reinterpret_cast<double2 *>(stage + lane * kSliceBytes + j * 16) = make_double2(v[2 * j], v[2 * j + 1]);
        __syncwarp();
#pragma unroll
        for (int k = 0; k < M / 2; ++k)
            *reinterpret_cast<double2 *>(grow + 2 * (k * 32 + lane)) =
                *reinterpret_cast<const double2 *>(stage + unit_offset(k * 32 + lane));
        __syncwarp();
    }
};
