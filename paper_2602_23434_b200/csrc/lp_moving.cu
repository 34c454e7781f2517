// lp_moving.cu -- spectral update on a per-particle moving energy grid (NEXT-5; readings E1-E4 of DESIGN.md
// section 3; the eng_ array of Listing 3; Eq. 6).
//
// Every particle carries its own N_b + 1 bin edges.  Over a step they follow the characteristics of Eq. 6,
//   eps' = alpha eps / (1 + beta eps),   alpha = e^{-s},  s = a dtau,  beta = c_r dtau (1 - e^{-s}) / s,
// and every bin keeps its number: chi_i' = chi_i dE_i / dE_i'.  With t_k = 1 + beta eps_k the new width is
// dE_i' = alpha dE_i / (t_i t_{i+1}) exactly, so chi_i' = chi_i t_i t_{i+1} / alpha -- no subtraction of nearly
// equal edges and one division per edge instead of two per bin.  No CFL limit and no substeps: the kernel is a
// pure stream of 16 (2 N_b + 1) bytes per particle behind a per-particle phase (gather, coefficients) that is
// the same as the fixed-grid kernel's (lp_spectral.cu).
//
// Staged (lp_spectral_update) or fused with the two push stages (lp_step), like the fixed-grid kernel.
// A block takes 128 particles at a time: phase 1 with one thread per particle leaves (alpha, beta) in shared
// memory, then its four warps stream the 128 rows, RI rows per warp in flight.  Several blocks are resident
// per SM, so the latency-bound phase of one overlaps the stream of the others.  sm_100a.
#include "lp_device.cuh"

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kThreads = 128;
constexpr int kWarps = kThreads / 32;

struct LpMovingArgs {
    LpGeom g;
    LpCells cells;
    double *x, *y, *z;           // staged: x^{n+1} (read only); fused: x^{n+1} out
    const double *xin, *yin, *zin;   // positions read (== x, y, z unless the step re-sorts)
    // Re-sort folded into the fused step (as in lp_spectral.cu): particle p of the new order is the one stored at
    // perm[p] of xin.., id_in, eng_in, chi_in; everything is written at p of the other buffer set.
    const uint32_t *perm;        // or NULL
    const uint64_t *id_in;
    uint64_t *id_out;
    const double *rho_old;       // staged: from push stage 0
    int32_t *status;             // fused: outside-box flags [np]
    const double *eng_in;        // [np][nbins + 1]
    double *eng;                 // [np][nbins + 1] out (== eng_in unless the step re-sorts)
    const double *chi_in;        // [np][nbins]
    double *chi;                 // [np][nbins] out
    int32_t *nsub_ws;            // [np]: 1 (one exact step per particle)
    int32_t *nsub_user;          // or NULL
    long long np;
    double dt, kappa, u_rad;
};

// per-particle phase: [FUSED: push stages a5, a6,] coefficients a7, then (alpha, beta) of the step (reading E2)
template <bool FUSED>
__device__ __forceinline__ double2 lp_moving_coef(const LpMovingArgs &A, long long p, double px, double py, double pz)
{
    double a, cr, dtau;
    lp_particle_coefficients<FUSED>(A.g, A.cells, A.dt, A.kappa, A.u_rad, A.x, A.y, A.z, A.status, A.rho_old, p, px, py, pz,
                                    a, cr, dtau);
    const double s = __dmul_rn(a, dtau);
    const double alpha = exp(-s);
    const double crt = __dmul_rn(cr, dtau);
    const double beta = (s != 0.0) ? __dmul_rn(crt, __ddiv_rn(-expm1(-s), s)) : crt;
    return make_double2(alpha, beta);
}

// Resident blocks per SM, staged kernel: six at N_b <= 64 (84 registers; the per-particle phase is a larger share
// of a short row and needs more blocks to hide behind), four above (measured: 64 bins 0.806 -> 0.828 of the copy
// bandwidth with six, 128 / 256 bins 0.89 / 0.90 -> 0.875 / 0.865; eight blocks or eight rows in flight lose
// everywhere).  The fused kernel (push stages in the per-particle phase: three stencils, the corner records kept
// in registers between them) gets four.  A warp-specialised variant (one particle warp working a group ahead of
// three row warps, a block barrier per group) was measured slower: 0.74 instead of 0.79 at 64 bins, 0.52 instead
// of 0.72 at 16.
// MODE: 0 staged (lp_spectral_update), 1 fused step, 2 fused step that re-sorts (reads through A.perm).
template <int NB, int MODE>
__global__ void __launch_bounds__(kThreads, (NB <= 64 && MODE == 0) ? 6 : 4) lp_moving_kernel(LpMovingArgs A)
{
    constexpr bool FUSED = MODE >= 1, PERM = MODE == 2;
    constexpr int G = NB < 32 ? NB : 32;         // lanes per row
    constexpr int PPW = 32 / G;                  // rows a warp holds side by side
    constexpr int M = NB / G;                    // bins per lane: bin sub + G j
    constexpr int RI = M <= 2 ? 4 : (M == 4 ? 2 : 1);      // row sets in flight per warp
    constexpr int ROWS = PPW * RI;               // rows per warp trip
    static_assert(32 % ROWS == 0 || ROWS <= 32, "rows per trip");

    __shared__ double2 sAB[kThreads];
    __shared__ uint32_t sSrc[PERM ? kThreads : 1];          // source row of every particle of the group
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane % G, grp = lane / G;
    const long long ngroups = (A.np + kThreads - 1) / kThreads;

    for (long long gidx = blockIdx.x; gidx < ngroups; gidx += gridDim.x) {
        const long long base = gidx * kThreads;
        {
            const long long p = base + threadIdx.x;
            double2 ab = make_double2(1.0, 0.0);
            if (p < A.np) {
                const size_t src = PERM ? (size_t)A.perm[p] : (size_t)p;
                if (PERM) {
                    sSrc[threadIdx.x] = (uint32_t)src;
                    A.id_out[p] = A.id_in[src];
                }
                ab = lp_moving_coef<FUSED>(A, p, A.xin[src], A.yin[src], A.zin[src]);
                __stcs(A.nsub_ws + p, 1);
                if (A.nsub_user) __stcs(A.nsub_user + p, 1);
            }
            sAB[threadIdx.x] = ab;
        }
        __syncthreads();
        // rows of this warp: base + warp*32 + [0, 32)
        for (int r0 = 0; r0 < 32; r0 += ROWS) {
            double e[RI][M], en[RI], c[RI][M];
            double2 ab[RI];
            long long row[RI];
            bool have[RI];
#pragma unroll
            for (int u = 0; u < RI; ++u) {
                const int rl = warp * 32 + r0 + u * PPW + grp;          // row within the block's 128
                row[u] = base + rl;
                have[u] = row[u] < A.np;
                ab[u] = sAB[rl];
                const long long srow = (PERM && have[u]) ? (long long)sSrc[rl] : row[u];
                const double *er = A.eng_in + srow * (NB + 1);
                const double *cp = A.chi_in + srow * NB;
#pragma unroll
                for (int j = 0; j < M; ++j) {
                    e[u][j] = have[u] ? __ldcs(er + sub + G * j) : 1.0;
                    c[u][j] = have[u] ? __ldcs(cp + sub + G * j) : 0.0;
                }
                en[u] = have[u] ? __ldcs(er + NB) : 1.0;               // the top edge (same address in the group)
            }
#pragma unroll
            for (int u = 0; u < RI; ++u) {
                const double alpha = ab[u].x, beta = ab[u].y;
                const double ralpha = 1.0 / alpha;
                double t[M], tn;
#pragma unroll
                for (int j = 0; j < M; ++j) t[j] = fma(beta, e[u][j], 1.0);
                tn = fma(beta, en[u], 1.0);
                double *er = A.eng + row[u] * (NB + 1);
                double *cp = A.chi + row[u] * NB;
#pragma unroll
                for (int j = 0; j < M; ++j) {
                    // t of the next edge: the next lane's, or (last lane of the group) the group's first lane
                    // one round further on, or the top edge
                    const double from_next = __shfl_down_sync(kFull, t[j], 1, G);
                    const double wrap = (j + 1 < M) ? __shfl_sync(kFull, t[(j + 1 < M) ? j + 1 : j], 0, G) : tn;
                    const double t_up = (sub == G - 1) ? wrap : from_next;
                    if (have[u]) {
                        __stcs(er + sub + G * j, alpha * e[u][j] / t[j]);
                        __stcs(cp + sub + G * j, c[u][j] * (t[j] * t_up) * ralpha);
                    }
                }
                if (have[u] && sub == 0) __stcs(er + NB, alpha * en[u] / tn);
            }
        }
        __syncthreads();                       // sAB is rewritten by the next group
    }
}

// eng rows [first, first + count) <- the fixed table's edges (reading E4)
__global__ void __launch_bounds__(256)
lp_moving_init_kernel(const double *__restrict__ tab, int nbins, double *__restrict__ eng, long long first, long long count)
{
    const long long n = count * (nbins + 1);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        eng[first * (nbins + 1) + i] = tab[i % (nbins + 1)];
}

// rows of `len` doubles through a permutation (rows may be 8-byte aligned only): a warp per row
__global__ void __launch_bounds__(256)
lp_permute_rows8_kernel(const uint32_t *__restrict__ perm, const double *__restrict__ src, double *__restrict__ dst,
                        long long np, int len)
{
    const int lane = threadIdx.x & 31;
    const long long gw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long r = gw; r < np; r += nw) {
        const double *s = src + (long long)perm[r] * len;
        double *d = dst + r * len;
        for (int i = lane; i < len; i += 32) __stcs(d + i, __ldcs(s + i));
    }
}

template <int NB, int MODE>
int launch_mode(const LpMovingArgs &a, int sm_count, cudaStream_t s)
{
    int per_sm = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lp_moving_kernel<NB, MODE>, kThreads, 0);
    if (per_sm < 1) per_sm = 1;
    const long long want = (a.np + kThreads - 1) / kThreads;
    const long long cap = (long long)sm_count * per_sm;
    int blocks = (int)(want < cap ? want : cap);
    if (blocks < 1) blocks = 1;
    lp_moving_kernel<NB, MODE><<<blocks, kThreads, 0, s>>>(a);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

template <int NB>
int launch(const LpMovingArgs &a, bool fused, int sm_count, cudaStream_t s)
{
    if (!fused) return launch_mode<NB, 0>(a, sm_count, s);
    return a.perm ? launch_mode<NB, 2>(a, sm_count, s) : launch_mode<NB, 1>(a, sm_count, s);
}

}  // namespace

int lp_launch_moving(const LpGeom &g, const LpCells &cells, const LpMovingIO &io, const double *rho_old, int32_t *status,
                     bool fused, int32_t *nsub_ws, int32_t *nsub_user, long long np, int nbins, double dt, double kappa,
                     double u_rad, int sm_count, cudaStream_t s)
{
    LpMovingArgs a;
    a.g = g; a.cells = cells;
    a.x = io.x; a.y = io.y; a.z = io.z;
    a.xin = io.xin; a.yin = io.yin; a.zin = io.zin;
    a.perm = io.perm; a.id_in = io.id_in; a.id_out = io.id_out;
    a.rho_old = rho_old;
    a.status = status;
    a.eng_in = io.eng_in; a.eng = io.eng;
    a.chi_in = io.chi_in; a.chi = io.chi;
    a.nsub_ws = nsub_ws; a.nsub_user = nsub_user;
    a.np = np;
    a.dt = dt; a.kappa = kappa; a.u_rad = u_rad;
    switch (nbins) {
    case 16:  return launch<16>(a, fused, sm_count, s);
    case 32:  return launch<32>(a, fused, sm_count, s);
    case 64:  return launch<64>(a, fused, sm_count, s);
    case 128: return launch<128>(a, fused, sm_count, s);
    case 256: return launch<256>(a, fused, sm_count, s);
    case 512: return launch<512>(a, fused, sm_count, s);
    default:  return -1;
    }
}

int lp_launch_moving_init(const double *tab, int nbins, double *eng, long long first, long long count, cudaStream_t s)
{
    if (count <= 0) return 0;
    long long blocks = (count * (nbins + 1) + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    lp_moving_init_kernel<<<(int)blocks, 256, 0, s>>>(tab, nbins, eng, first, count);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int lp_launch_permute_rows8(const uint32_t *perm, const double *src, double *dst, long long np, int len, cudaStream_t s)
{
    long long blocks = (np + 7) / 8;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (blocks < 1) blocks = 1;
    lp_permute_rows8_kernel<<<(int)blocks, 256, 0, s>>>(perm, src, dst, np, len);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}
