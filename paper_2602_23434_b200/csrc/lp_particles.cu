// lp_particles.cu -- field repack, cell key + trilinear gather, two-stage push (thread per particle).
// Steps a1, a3-a6 of DESIGN.md section 1.  sm_100a.
#include "lp_device.cuh"

namespace {

constexpr int kThreads = 256;

inline int blocks_for(long long n, int threads)
{
    long long b = (n + threads - 1) / threads;
    return (int)(b < 1 ? 1 : b);
}

// a3: seven SoA grid arrays -> one 64-byte record per cell, written as its two 32-byte halves.
__global__ void __launch_bounds__(kThreads)
lp_repack_kernel(const double *__restrict__ vx, const double *__restrict__ vy, const double *__restrict__ vz,
                 const double *__restrict__ bx, const double *__restrict__ by, const double *__restrict__ bz,
                 const double *__restrict__ rho, double4 *__restrict__ recA, double4 *__restrict__ recB,
                 unsigned stride, long long ncell)
{
    long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    double2 *a = reinterpret_cast<double2 *>(recA + (size_t)stride * c);
    double2 *b = reinterpret_cast<double2 *>(recB + (size_t)stride * c);
    a[0] = make_double2(vx[c], vy[c]);
    a[1] = make_double2(vz[c], rho[c]);
    b[0] = make_double2(bx[c], by[c]);
    b[1] = make_double2(bz[c], 0.0);
}

// a1 + a4: key and/or the seven sampled fields at the current positions.
__global__ void __launch_bounds__(kThreads)
lp_interpolate_kernel(LpGeom g, LpCells cells, const double *__restrict__ x, const double *__restrict__ y,
                      const double *__restrict__ z, long long np, double *__restrict__ out7,
                      uint32_t *__restrict__ key)
{
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    double px = x[p], py = y[p], pz = z[p];
    if (key) key[p] = lp_cell_key(g, px, py, pz);
    if (out7) {
        LpStencil st;
        lp_stencil(g, px, py, pz, st);
        double a[4], b[3];
        lp_gather_A(cells, st, a);
        lp_gather_B(cells, st, b);
        out7[p] = a[0];
        out7[np + p] = a[1];
        out7[2 * np + p] = a[2];
        out7[3 * np + p] = b[0];
        out7[4 * np + p] = b[1];
        out7[5 * np + p] = b[2];
        out7[6 * np + p] = a[3];
    }
}

// a4 through shared-memory tiles, for particle sets sorted by cell (the option north_star names next to the direct
// gather; measured against it in profiles/r02_gather_tile.md).  A block of kTileBlock consecutive particles finds
// the bounding box of its stencils (in unwrapped cell indices, so a box may straddle a periodic seam), loads the
// box's cell records once, coalesced, and every particle gathers its eight corners from shared memory with the
// same weights in the same order as the direct path: bit-identical values.  A box that does not fit (particles
// not sorted, or drifted far apart) falls back to the direct gather for that block.
constexpr int kTileBlock = 64;

__device__ __forceinline__ void lp_axis_raw(double x, double lo, double inv_dx, int &b, double &w0, double &w1)
{
    const double s = __dsub_rn(__dmul_rn(__dsub_rn(x, lo), inv_dx), 0.5);
    const double fl = floor(s);
    const double f = __dsub_rn(s, fl);
    // clamp far-away positions so that the int conversion is defined; such a block takes the direct path
    b = (int)fmin(fmax(fl, -1.0e9), 1.0e9);
    w0 = __dsub_rn(1.0, f);
    w1 = f;
}

__global__ void __launch_bounds__(kTileBlock)
lp_interpolate_tile_kernel(LpGeom g, LpCells cells, const double *__restrict__ x, const double *__restrict__ y,
                           const double *__restrict__ z, long long np, double *__restrict__ out7, int max_cells)
{
    extern __shared__ __align__(32) unsigned char lp_tile_raw[];
    LpRec *tile = reinterpret_cast<LpRec *>(lp_tile_raw);          // [cell][A | B]
    __shared__ int smin[3][kTileBlock / 32], smax[3][kTileBlock / 32];

    const long long p = (long long)blockIdx.x * kTileBlock + threadIdx.x;
    const bool valid = p < np;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int b[3] = { 0, 0, 0 };
    double w[3][2] = { { 1.0, 0.0 }, { 1.0, 0.0 }, { 1.0, 0.0 } };
    double px = 0.0, py = 0.0, pz = 0.0;
    if (valid) {
        px = x[p]; py = y[p]; pz = z[p];
        lp_axis_raw(px, g.xlo[0], g.inv_dx[0], b[0], w[0][0], w[0][1]);
        lp_axis_raw(py, g.xlo[1], g.inv_dx[1], b[1], w[1][0], w[1][1]);
        lp_axis_raw(pz, g.xlo[2], g.inv_dx[2], b[2], w[2][0], w[2][1]);
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int lo = __reduce_min_sync(0xffffffffu, valid ? b[d] : 0x7fffffff);
        const int hi = __reduce_max_sync(0xffffffffu, valid ? b[d] : (int)0x80000000);
        if (lane == 0) { smin[d][warp] = lo; smax[d][warp] = hi; }
    }
    __syncthreads();
    int lo3[3], ext[3];
    long long ncell = 1;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        int lo = smin[d][0], hi = smax[d][0];
#pragma unroll
        for (int k = 1; k < kTileBlock / 32; ++k) { lo = min(lo, smin[d][k]); hi = max(hi, smax[d][k]); }
        lo3[d] = lo;
        ext[d] = (hi >= lo) ? (int)min((long long)hi - lo + 2, 1ll << 20) : 0;
        ncell *= ext[d];
    }
    double a[4], bb[3];
    if (ncell > 0 && ncell <= max_cells) {                        // (uniform over the block)
        const int n3[3] = { g.nx, g.ny, g.nz };
        // a warp takes whole x-rows of the box: consecutive lanes read consecutive records
        for (int row = warp; row < ext[1] * ext[2]; row += kTileBlock / 32) {
            const int iy = row % ext[1], iz = row / ext[1];
            const int cj = lp_wrap(lo3[1] + iy, n3[1], g.per[1]);
            const int ck = lp_wrap(lo3[2] + iz, n3[2], g.per[2]);
            for (int ix = lane; ix < ext[0]; ix += 32) {
                const int ci = lp_wrap(lo3[0] + ix, n3[0], g.per[0]);
                const size_t cell = (size_t)((ck * g.ny + cj) * g.nx + ci);
                const int c = row * ext[0] + ix;
                tile[2 * c] = lp_ldg_rec(cells.recA + (size_t)cells.stride * cell);
                tile[2 * c + 1] = lp_ldg_rec(cells.recB + (size_t)cells.stride * cell);
            }
        }
        __syncthreads();
        if (valid) {
            a[0] = a[1] = a[2] = a[3] = 0.0;
            bb[0] = bb[1] = bb[2] = 0.0;
            const int ox = b[0] - lo3[0], oy = b[1] - lo3[1], oz = b[2] - lo3[2];
#pragma unroll
            for (int cz = 0; cz < 2; ++cz)
#pragma unroll
                for (int cy = 0; cy < 2; ++cy)
#pragma unroll
                    for (int cx = 0; cx < 2; ++cx) {
                        const double wt = __dmul_rn(__dmul_rn(w[2][cz], w[1][cy]), w[0][cx]);
                        const int c = ((oz + cz) * ext[1] + (oy + cy)) * ext[0] + (ox + cx);
                        const LpRec ra = tile[2 * c], rb = tile[2 * c + 1];
                        a[0] = lp_acc(a[0], wt, ra.a); a[1] = lp_acc(a[1], wt, ra.b);
                        a[2] = lp_acc(a[2], wt, ra.c); a[3] = lp_acc(a[3], wt, ra.d);
                        bb[0] = lp_acc(bb[0], wt, rb.a); bb[1] = lp_acc(bb[1], wt, rb.b); bb[2] = lp_acc(bb[2], wt, rb.c);
                    }
        }
    } else if (valid) {
        LpStencil st;
        lp_stencil(g, px, py, pz, st);
        lp_gather_A(cells, st, a);
        lp_gather_B(cells, st, bb);
    }
    if (valid) {
        out7[p] = a[0];
        out7[np + p] = a[1];
        out7[2 * np + p] = a[2];
        out7[3 * np + p] = bb[0];
        out7[4 * np + p] = bb[1];
        out7[5 * np + p] = bb[2];
        out7[6 * np + p] = a[3];
    }
}

// a5: k1 = v(x^n), rho_old = rho(x^n), x* = x^n + dt*k1
__global__ void __launch_bounds__(kThreads) lp_push0_kernel(LpPushArgs A)
{
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= A.np) return;
    double px = A.x[p], py = A.y[p], pz = A.z[p];
    LpStencil st;
    lp_stencil(A.g, px, py, pz, st);
    double q[4];
    lp_gather_A(A.cells, st, q);
    const long long np = A.np;
    A.k1[p] = q[0];
    A.k1[np + p] = q[1];
    A.k1[2 * np + p] = q[2];
    A.rho_old[p] = q[3];
    A.xs[p] = __dadd_rn(px, __dmul_rn(A.dt, q[0]));
    A.xs[np + p] = __dadd_rn(py, __dmul_rn(A.dt, q[1]));
    A.xs[2 * np + p] = __dadd_rn(pz, __dmul_rn(A.dt, q[2]));
}

// a6: x^{n+1} = x^n + (dt/2)(k1 + v(x*)), periodic wrap / outside flag
__global__ void __launch_bounds__(kThreads) lp_push1_kernel(LpPushArgs A)
{
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= A.np) return;
    const long long np = A.np;
    LpStencil st;
    lp_stencil(A.g, A.xs[p], A.xs[np + p], A.xs[2 * np + p], st);
    double k2[3];
    lp_gather_v(A.cells, st, k2);
    const double hdt = __dmul_rn(0.5, A.dt);
    double *pos[3] = { A.x, A.y, A.z };
    int stt = 0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double xn = __dadd_rn(pos[d][p], __dmul_rn(hdt, __dadd_rn(A.k1[(long long)d * np + p], k2[d])));
        if (A.g.per[d]) xn = lp_wrap_pos(xn, A.g.xlo[d], A.g.xhi[d], A.g.len[d]);
        else if (xn < A.g.xlo[d] || xn >= A.g.xhi[d]) stt |= (1 << d);
        pos[d][p] = xn;
    }
    A.status[p] = stt;
}

// Three-stage third-order pusher (reading K1 of DESIGN.md), one launch per stage:
//   0: x0 = x^n kept in the x* scratch, rho_old = rho(x^n), x <- x0 + dt v(x0)
//   1: x <- (3/4) x0 + (1/4) (x + dt v(x))
//   2: x <- (x0 + 2 (x + dt v(x))) / 3, periodic wrap / outside flag
template <int STAGE>
__global__ void __launch_bounds__(kThreads) lp_push_rk3_kernel(LpPushArgs A)
{
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= A.np) return;
    const long long np = A.np;
    double *pos[3] = { A.x, A.y, A.z };
    const double cur[3] = { A.x[p], A.y[p], A.z[p] };
    LpStencil st;
    lp_stencil(A.g, cur[0], cur[1], cur[2], st);
    double q[4];
    lp_gather_A(A.cells, st, q);
    int stt = 0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double adv = __dadd_rn(cur[d], __dmul_rn(A.dt, q[d]));
        double xn;
        if (STAGE == 0) {
            A.xs[(long long)d * np + p] = cur[d];
            xn = adv;
        } else if (STAGE == 1) {
            xn = __dadd_rn(__dmul_rn(0.75, A.xs[(long long)d * np + p]), __dmul_rn(0.25, adv));
        } else {
            xn = __ddiv_rn(__dadd_rn(A.xs[(long long)d * np + p], __dmul_rn(2.0, adv)), 3.0);
            if (A.g.per[d]) xn = lp_wrap_pos(xn, A.g.xlo[d], A.g.xhi[d], A.g.len[d]);
            else if (xn < A.g.xlo[d] || xn >= A.g.xhi[d]) stt |= (1 << d);
        }
        pos[d][p] = xn;
    }
    if (STAGE == 0) A.rho_old[p] = q[3];
    if (STAGE == 2) A.status[p] = stt;
}

}  // namespace

int lp_launch_push_rk3(const LpPushArgs &a, int stage, cudaStream_t s)
{
    const int blocks = blocks_for(a.np, kThreads);
    if (stage == 0) lp_push_rk3_kernel<0><<<blocks, kThreads, 0, s>>>(a);
    else if (stage == 1) lp_push_rk3_kernel<1><<<blocks, kThreads, 0, s>>>(a);
    else lp_push_rk3_kernel<2><<<blocks, kThreads, 0, s>>>(a);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int lp_launch_repack(const double *const f[7], double4 *recA, double4 *recB, unsigned stride, long long ncell,
                     cudaStream_t s)
{
    lp_repack_kernel<<<blocks_for(ncell, kThreads), kThreads, 0, s>>>(f[0], f[1], f[2], f[3], f[4], f[5], f[6],
                                                                      recA, recB, stride, ncell);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int lp_launch_interpolate(const LpGeom &g, const LpCells &c, const double *x, const double *y, const double *z,
                          long long np, double *out7, uint32_t *key, cudaStream_t s)
{
    lp_interpolate_kernel<<<blocks_for(np, kThreads), kThreads, 0, s>>>(g, c, x, y, z, np, out7, key);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int lp_launch_interpolate_tiled(const LpGeom &g, const LpCells &c, const double *x, const double *y, const double *z,
                                long long np, double *out7, bool *configured, cudaStream_t s)
{
    constexpr int kMaxCells = 384;                               // 24 KB of records per block: nine blocks per SM
    const size_t smem = (size_t)kMaxCells * 64;
    if (!*configured) {                                          // once per context (a context lives on one device)
        if (cudaFuncSetAttribute(lp_interpolate_tile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
        *configured = true;
    }
    lp_interpolate_tile_kernel<<<blocks_for(np, kTileBlock), kTileBlock, smem, s>>>(g, c, x, y, z, np, out7, kMaxCells);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int lp_launch_push0(const LpPushArgs &a, cudaStream_t s)
{
    lp_push0_kernel<<<blocks_for(a.np, kThreads), kThreads, 0, s>>>(a);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int lp_launch_push1(const LpPushArgs &a, cudaStream_t s)
{
    lp_push1_kernel<<<blocks_for(a.np, kThreads), kThreads, 0, s>>>(a);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}
