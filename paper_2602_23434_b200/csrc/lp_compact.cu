// lp_compact.cu -- deletion of flagged particles with hole filling (reading C1 of
// DESIGN.md section 3): the N_del flagged particles go, the survivors stored at i >= N_p - N_del ("fillers")
// move into the flagged slots below N_p - N_del ("holes"), k-th hole (ascending) <- k-th filler (ascending).
//
// One exclusive prefix sum of the flags gives every index its rank among the flagged ones:
//   hole number of a flagged i < keep      = rank[i]                       (every flagged index before it is a hole too)
//   filler number of an unflagged i >= keep = (i - keep) - (rank[i] - rank[keep])
// so holes and fillers are listed without a second compaction, and the move is one gather/scatter over
// H = rank[keep] particles (their x, y, z, id and chi rows).  The paper's two cycles over N_p and one over
// N_del, one over N_f are the count, the rank pass, and the move.  sm_100a.
#include "lp_internal.h"

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kItems = 16;
constexpr int kTile = kThreads * kItems;          // flags per block

inline int blocks_for(long long n, int per) { long long b = (n + per - 1) / per; return (int)(b < 1 ? 1 : b); }

// block-wide exclusive scan of one value per thread; returns the exclusive prefix, total in *total
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t *total)
{
    __shared__ uint32_t wsum[kWarps];
    __shared__ uint32_t tot;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t u = __shfl_up_sync(kFull, inc, o);
        if (lane >= o) inc += u;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    uint32_t wbase = 0;
    for (int w = 0; w < warp; ++w) wbase += wsum[w];
    if (threadIdx.x == kThreads - 1) tot = wbase + inc;
    __syncthreads();
    *total = tot;
    const uint32_t r = wbase + inc - v;
    __syncthreads();                                // wsum / tot may be reused by the next call
    return r;
}

// step 1a: flags of a tile (thread t owns items t*kItems .. +kItems, so ranks follow the index order)
__global__ void __launch_bounds__(kThreads)
lp_flag_count_kernel(const int32_t *__restrict__ flag, long long np, uint32_t *__restrict__ blk)
{
    const long long i0 = (long long)blockIdx.x * kTile + (long long)threadIdx.x * kItems;
    uint32_t c = 0;
#pragma unroll
    for (int k = 0; k < kItems; ++k)
        if (i0 + k < np && flag[i0 + k] != 0) ++c;
    uint32_t total;
    block_excl_scan(c, &total);
    if (threadIdx.x == 0) blk[blockIdx.x] = total;
}

// step 1b: exclusive scan of the block counts (one block), N_del into counts[0]
__global__ void __launch_bounds__(kThreads)
lp_flag_scan_kernel(uint32_t *__restrict__ blk, int nblocks, unsigned long long *__restrict__ counts)
{
    uint32_t carry = 0;
    for (int b0 = 0; b0 < nblocks; b0 += kThreads) {
        const int i = b0 + threadIdx.x;
        const uint32_t v = i < nblocks ? blk[i] : 0u;
        uint32_t total;
        const uint32_t ex = block_excl_scan(v, &total);
        if (i < nblocks) blk[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0) counts[0] = carry;
}

// rank[i] = flagged indices below i
__global__ void __launch_bounds__(kThreads)
lp_flag_rank_kernel(const int32_t *__restrict__ flag, long long np, const uint32_t *__restrict__ blk,
                    uint32_t *__restrict__ rank)
{
    const long long i0 = (long long)blockIdx.x * kTile + (long long)threadIdx.x * kItems;
    uint32_t f[kItems], c = 0;
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        f[k] = (i0 + k < np && flag[i0 + k] != 0) ? 1u : 0u;
        c += f[k];
    }
    uint32_t total;
    uint32_t run = blk[blockIdx.x] + block_excl_scan(c, &total);
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        if (i0 + k < np) rank[i0 + k] = run;
        run += f[k];
    }
}

// steps 2 and 3: the holes and the fillers, each in ascending order; counts[1] = H
__global__ void __launch_bounds__(kThreads)
lp_holes_fillers_kernel(const int32_t *__restrict__ flag, const uint32_t *__restrict__ rank, long long np,
                        unsigned long long *__restrict__ counts, uint32_t *__restrict__ hole,
                        uint32_t *__restrict__ filler)
{
    const long long keep = np - (long long)counts[0];
    const uint32_t h = keep < np ? rank[keep] : (uint32_t)counts[0];      // flagged below the cut
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) counts[1] = h;
    if (i >= np) return;
    const bool del = flag[i] != 0;
    if (i < keep) {
        if (del) hole[rank[i]] = (uint32_t)i;
    } else if (!del) {
        filler[(uint32_t)(i - keep) - (rank[i] - h)] = (uint32_t)i;
    }
}

// step 4: every parameter of filler k into hole k (a warp per particle: the row in 16-byte pieces)
__global__ void __launch_bounds__(kThreads)
lp_fill_holes_kernel(const unsigned long long *__restrict__ counts, const uint32_t *__restrict__ hole,
                     const uint32_t *__restrict__ filler, double *__restrict__ x, double *__restrict__ y,
                     double *__restrict__ z, uint64_t *__restrict__ id, double *__restrict__ chi, int nbins,
                     double *__restrict__ eng /*[np][nbins+1] or NULL*/)
{
    const long long h = (long long)counts[1];
    const int lane = threadIdx.x & 31;
    const long long gw = ((long long)blockIdx.x * kThreads + threadIdx.x) >> 5;
    const long long nw = ((long long)gridDim.x * kThreads) >> 5;
    for (long long k = gw; k < h; k += nw) {
        const long long d = hole[k], s = filler[k];
        if (lane == 0) { x[d] = x[s]; y[d] = y[s]; z[d] = z[s]; id[d] = id[s]; }
        const double2 *src = reinterpret_cast<const double2 *>(chi + s * nbins);
        double2 *dst = reinterpret_cast<double2 *>(chi + d * nbins);
        for (int i = lane; i < nbins / 2; i += 32) dst[i] = src[i];
        if (eng)            // the particle's energy-grid row (8-byte aligned only)
            for (int i = lane; i <= nbins; i += 32) eng[d * (nbins + 1) + i] = eng[s * (nbins + 1) + i];
    }
}

inline bool ok() { return cudaPeekAtLastError() == cudaSuccess; }

}  // namespace

size_t lp_compact_block_elems(long long np) { return (size_t)blocks_for(np, kTile) + 1; }

// counts: 2 x u64 on the device (N_del, H).  Returns kernels launched or -1.
int lp_launch_compact(const int32_t *flag, long long np, int nbins, uint32_t *blk, uint32_t *rank, uint32_t *hole,
                      uint32_t *filler, unsigned long long *counts, double *x, double *y, double *z, uint64_t *id,
                      double *chi, double *eng, int sm_count, cudaStream_t s)
{
    const int nblocks = blocks_for(np, kTile);
    lp_flag_count_kernel<<<nblocks, kThreads, 0, s>>>(flag, np, blk);
    lp_flag_scan_kernel<<<1, kThreads, 0, s>>>(blk, nblocks, counts);
    lp_flag_rank_kernel<<<nblocks, kThreads, 0, s>>>(flag, np, blk, rank);
    lp_holes_fillers_kernel<<<blocks_for(np, kThreads), kThreads, 0, s>>>(flag, rank, np, counts, hole, filler);
    long long fb = (np + kWarps - 1) / kWarps;
    const long long cap = (long long)sm_count * 8;
    if (fb > cap) fb = cap;
    if (fb < 1) fb = 1;
    lp_fill_holes_kernel<<<(int)fb, kThreads, 0, s>>>(counts, hole, filler, x, y, z, id, chi, nbins, eng);
    return ok() ? 5 : -1;
}
