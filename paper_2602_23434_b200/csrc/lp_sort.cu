// lp_sort.cu -- step a2 of DESIGN.md section 1: order particles ascending by (cell key, id) and
// apply the permutation.  A stable LSD radix sort (8-bit digits) over a u32 index array: first the
// digits of id, then the digits of the cell key, so ties in the key keep ascending id.  Stability
// and the unique ids make the result the one total order the oracle's comparison sort produces.
// Also: the aggregate diagnostics reduction (a10).  sm_100a.
#include "lp_device.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kItems = 16;                       // rounds per tile
constexpr int kTile = kThreads * kItems;         // elements per block
constexpr unsigned kFull = 0xffffffffu;

inline int blocks_for(long long n, int per) { long long b = (n + per - 1) / per; return (int)(b < 1 ? 1 : b); }

__global__ void __launch_bounds__(kThreads)
lp_key_kernel(LpGeom g, const double *__restrict__ x, const double *__restrict__ y,
              const double *__restrict__ z, long long np, uint32_t *__restrict__ key)
{
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < np) key[p] = lp_cell_key(g, x[p], y[p], z[p]);
}

// digit of element e of the current sequence (idx_in == NULL means the identity sequence)
__device__ __forceinline__ uint32_t lp_digit(const uint32_t *idx_in, const uint64_t *id, const uint32_t *key,
                                             long long e, int use_key, int shift, uint32_t &src)
{
    src = idx_in ? idx_in[e] : (uint32_t)e;
    return use_key ? ((key[src] >> shift) & 255u) : (uint32_t)((id[src] >> shift) & 255ull);
}

__global__ void __launch_bounds__(kThreads)
lp_radix_hist_kernel(const uint32_t *__restrict__ idx_in, const uint64_t *__restrict__ id,
                     const uint32_t *__restrict__ key, long long np, int use_key, int shift,
                     uint32_t *__restrict__ hist, int nblocks, uint8_t *__restrict__ digit,
                     const uint32_t *__restrict__ enable)
{
    if (enable && *enable == 0) return;          // fallback of the counting sort, not needed this time
    __shared__ uint32_t sh[256];
    sh[threadIdx.x] = 0;
    __syncthreads();
    const long long t0 = (long long)blockIdx.x * kTile;
    for (int r = 0; r < kItems; ++r) {
        long long e = t0 + r * kThreads + threadIdx.x;
        if (e < np) {
            uint32_t src;
            const uint32_t d = lp_digit(idx_in, id, key, e, use_key, shift, src);
            digit[e] = (uint8_t)d;              // kept for the scatter pass: one gather through the permutation, not two
            atomicAdd(&sh[d], 1u);
        }
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * nblocks + blockIdx.x] = sh[threadIdx.x];
}

// Per-digit exclusive scan over blocks: block d scans hist[d][0..nblocks) in place and writes the
// digit total to totals[d].  The scatter kernel adds the exclusive prefix of the totals itself.
__global__ void __launch_bounds__(kThreads)
lp_scan_rows_kernel(uint32_t *__restrict__ hist, int nblocks, uint32_t *__restrict__ totals,
                    const uint32_t *__restrict__ enable)
{
    if (enable && *enable == 0) return;
    __shared__ uint32_t wsum[kWarps];
    __shared__ uint32_t carry_s;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    uint32_t *row = hist + (size_t)blockIdx.x * nblocks;
    if (t == 0) carry_s = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nblocks; b0 += kThreads) {
        const int i = b0 + t;
        const uint32_t v = i < nblocks ? row[i] : 0u;
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
        const uint32_t carry = carry_s;
        if (i < nblocks) row[i] = carry + wbase + inc - v;
        __syncthreads();
        if (t == kThreads - 1) carry_s = carry + wbase + inc;
        __syncthreads();
    }
    if (t == 0) totals[blockIdx.x] = carry_s;
}

__global__ void __launch_bounds__(kThreads)
lp_radix_scatter_kernel(const uint32_t *__restrict__ idx_in, const uint64_t *__restrict__ id,
                        const uint32_t *__restrict__ key, long long np, int use_key, int shift,
                        const uint32_t *__restrict__ hist, const uint32_t *__restrict__ totals, int nblocks,
                        uint32_t *__restrict__ idx_out, const uint8_t *__restrict__ digit,
                        const uint32_t *__restrict__ enable)
{
    if (enable && *enable == 0) return;
    __shared__ uint32_t base[256];
    __shared__ uint32_t wcount[kWarps][256];
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    {   // exclusive prefix of the 256 digit totals (256 threads, one digit each)
        const uint32_t v = totals[t];
        uint32_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t u = __shfl_up_sync(kFull, inc, o);
            if (lane >= o) inc += u;
        }
        if (lane == 31) base[warp] = inc;
        __syncthreads();
        uint32_t wbase = 0;
        for (int w = 0; w < warp; ++w) wbase += base[w];
        __syncthreads();
        base[t] = wbase + inc - v + hist[(size_t)t * nblocks + blockIdx.x];
    }
    const long long t0 = (long long)blockIdx.x * kTile;
    for (int r = 0; r < kItems; ++r) {
#pragma unroll
        for (int w = 0; w < kWarps; ++w) wcount[w][t] = 0;
        __syncthreads();
        const long long e = t0 + r * kThreads + t;
        const bool valid = e < np;
        uint32_t src = 0, d = 256u + lane;          // invalid lanes get distinct pseudo-digits
        if (valid) {
            src = idx_in ? idx_in[e] : (uint32_t)e;
            d = digit[e];                        // written by lp_radix_hist_kernel of this pass
        }
        const unsigned same = __match_any_sync(kFull, d);
        const int rank = __popc(same & ((1u << lane) - 1u));
        if (valid && rank == 0) wcount[warp][d] = __popc(same);
        __syncthreads();
        {
            uint32_t run = base[t];
#pragma unroll
            for (int w = 0; w < kWarps; ++w) { uint32_t c = wcount[w][t]; wcount[w][t] = run; run += c; }
            base[t] = run;
        }
        __syncthreads();
        if (valid) idx_out[wcount[warp][d] + rank] = src;
        __syncthreads();
    }
}

// ---- counting sort by cell (the usual path): the key space is the grid, so one counter per cell orders the
// particles by key in O(N_p + cells) -- no radix passes -- and the few particles that share a cell are put in
// id order by rank counting inside their cell's segment.  The result is the same total (key, id) order.
//   K1 count:  key[p]; rank0[p] = atomicAdd(&cnt[key[p]], 1)        (arrival order inside the cell, arbitrary)
//   scan:      cnt -> exclusive offsets (cnt[ncell] = N_p)
//   K3 place:  seg_id[offset[key[p]] + rank0[p]] = id[p]            (the ids of a cell, contiguous)
//   K4 rank:   r = #{ids of my cell's segment smaller than mine};  perm[offset + r] = p
// A cell with more than kMaxSeg particles would make K4 quadratic: it raises *overflow instead and the radix
// passes (launched behind, every kernel gated on that flag) redo the whole sort.
constexpr int kMaxSeg = 64;

__global__ void __launch_bounds__(kThreads)
lp_cell_count_kernel(LpGeom g, const double *__restrict__ x, const double *__restrict__ y,
                     const double *__restrict__ z, long long np, uint32_t *__restrict__ key,
                     uint32_t *__restrict__ cnt, uint32_t *__restrict__ rank0)
{
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const uint32_t k = lp_cell_key(g, x[p], y[p], z[p]);
    key[p] = k;
    rank0[p] = atomicAdd(cnt + k, 1u);
}

// exclusive scan of v[0..n) in place, v[n] = total: tile sums, scan of the tile sums (one block), tiles again
constexpr int kScanItems = 16;
constexpr int kScanTile = kThreads * kScanItems;

__device__ __forceinline__ uint32_t lp_block_excl_scan(uint32_t v, uint32_t *total)
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
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(kThreads)
lp_scan_tile_sums_kernel(const uint32_t *__restrict__ v, long long n, uint32_t *__restrict__ tile_sum)
{
    const long long i0 = (long long)blockIdx.x * kScanTile + (long long)threadIdx.x * kScanItems;
    uint32_t c = 0;
    if (i0 + kScanItems <= n) {
        const uint4 *q = reinterpret_cast<const uint4 *>(v + i0);
#pragma unroll
        for (int k = 0; k < kScanItems / 4; ++k) { const uint4 t = q[k]; c += t.x + t.y + t.z + t.w; }
    } else {
        for (int k = 0; k < kScanItems; ++k) if (i0 + k < n) c += v[i0 + k];
    }
    uint32_t total;
    lp_block_excl_scan(c, &total);
    if (threadIdx.x == 0) tile_sum[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kThreads)
lp_scan_tile_offsets_kernel(uint32_t *__restrict__ tile_sum, int ntiles)
{
    uint32_t carry = 0;
    for (int b0 = 0; b0 < ntiles; b0 += kThreads) {
        const int i = b0 + threadIdx.x;
        const uint32_t v = i < ntiles ? tile_sum[i] : 0u;
        uint32_t total;
        const uint32_t ex = lp_block_excl_scan(v, &total);
        if (i < ntiles) tile_sum[i] = carry + ex;
        carry += total;
    }
}

__global__ void __launch_bounds__(kThreads)
lp_scan_tiles_kernel(uint32_t *__restrict__ v, long long n, const uint32_t *__restrict__ tile_off)
{
    const long long i0 = (long long)blockIdx.x * kScanTile + (long long)threadIdx.x * kScanItems;
    uint32_t f[kScanItems], c = 0;
    const bool full = i0 + kScanItems <= n;
    if (full) {
        const uint4 *q = reinterpret_cast<const uint4 *>(v + i0);
#pragma unroll
        for (int k = 0; k < kScanItems / 4; ++k) {
            const uint4 t = q[k];
            f[4 * k] = t.x; f[4 * k + 1] = t.y; f[4 * k + 2] = t.z; f[4 * k + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) f[k] = i0 + k < n ? v[i0 + k] : 0u;
    }
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) c += f[k];
    uint32_t total;
    uint32_t run = tile_off[blockIdx.x] + lp_block_excl_scan(c, &total);
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) { const uint32_t t = f[k]; f[k] = run; run += t; }
    if (full) {
        uint4 *q = reinterpret_cast<uint4 *>(v + i0);
#pragma unroll
        for (int k = 0; k < kScanItems / 4; ++k) q[k] = make_uint4(f[4 * k], f[4 * k + 1], f[4 * k + 2], f[4 * k + 3]);
    } else {
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) if (i0 + k < n) v[i0 + k] = f[k];
    }
    // the total behind the last element: the tile that holds index n - 1 writes v[n]
    if (i0 <= n - 1 && n - 1 < i0 + kScanItems) v[n] = run;
}

__global__ void __launch_bounds__(kThreads)
lp_cell_place_kernel(const uint32_t *__restrict__ key, const uint32_t *__restrict__ rank0,
                     const uint32_t *__restrict__ off, const uint64_t *__restrict__ id, long long np,
                     uint64_t *__restrict__ seg_id)
{
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    seg_id[off[key[p]] + rank0[p]] = id[p];
}

__global__ void __launch_bounds__(kThreads)
lp_cell_rank_kernel(const uint32_t *__restrict__ key, const uint32_t *__restrict__ off,
                    const uint64_t *__restrict__ id, const uint64_t *__restrict__ seg_id, long long np,
                    uint32_t *__restrict__ perm, uint32_t *__restrict__ overflow)
{
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const uint32_t k = key[p];
    const uint32_t o = off[k], n = off[k + 1] - o;
    uint32_t r = 0;
    if (n > 1) {
        if (n > (uint32_t)kMaxSeg) { *overflow = 1u; return; }
        const uint64_t mine = id[p];
        uint32_t same = 0;
        for (uint32_t j = 0; j < n; ++j) {
            const uint64_t other = seg_id[o + j];
            r += other < mine ? 1u : 0u;
            same += other == mine ? 1u : 0u;
        }
        // ids are unique by contract (lp.h).  Two equal ids in one cell would get the same rank, write one slot of
        // perm twice and leave another stale: hand such a set to the radix passes instead, which are stable (equal
        // (key, id) pairs stay in index order) -- a caller's bug then costs time, not a particle.
        if (same > 1) { *overflow = 1u; return; }
    }
    perm[o + r] = (uint32_t)p;
}

__global__ void __launch_bounds__(kThreads)
lp_copy_if_kernel(const uint32_t *__restrict__ src, uint32_t *__restrict__ dst, long long n,
                  const uint32_t *__restrict__ enable)
{
    if (*enable == 0) return;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        dst[i] = src[i];
}

__global__ void __launch_bounds__(kThreads)
lp_permute_f64_kernel(const uint32_t *__restrict__ perm, const double *__restrict__ src,
                      double *__restrict__ dst, long long np)
{
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < np) __stcs(dst + p, src[perm[p]]);
}

__global__ void __launch_bounds__(kThreads)
lp_permute_u64_kernel(const uint32_t *__restrict__ perm, const uint64_t *__restrict__ src,
                      uint64_t *__restrict__ dst, long long np)
{
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < np) __stcs(dst + p, src[perm[p]]);
}

// one warp (or half warp for 16 bins) moves one row of nbins doubles with 16-byte accesses
__global__ void __launch_bounds__(kThreads)
lp_permute_rows_kernel(const uint32_t *__restrict__ perm, const double *__restrict__ src,
                       double *__restrict__ dst, long long np, int nbins)
{
    const int lanes = nbins / 2 < 32 ? nbins / 2 : 32;      // lanes per row (16 B each per pass)
    const int rows_per_warp = 32 / lanes;
    const int lane = threadIdx.x & 31;
    const long long gw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nw = ((long long)gridDim.x * blockDim.x) >> 5;
    const int sub = lane % lanes, grp = lane / lanes;
    for (long long r0 = gw * rows_per_warp; r0 < np; r0 += nw * rows_per_warp) {
        const long long r = r0 + grp;
        if (r >= np) continue;
        const double2 *s = reinterpret_cast<const double2 *>(src + (long long)perm[r] * nbins);
        double2 *d = reinterpret_cast<double2 *>(dst + r * nbins);
        for (int i = sub; i < nbins / 2; i += lanes) __stcs(d + i, __ldcs(s + i));      // touched once: streaming
    }
}

__global__ void __launch_bounds__(kThreads)
lp_max_u64_kernel(const uint64_t *__restrict__ v, long long np, unsigned long long *out)
{
    unsigned long long m = 0;
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < np; p += (long long)gridDim.x * blockDim.x)
        m = v[p] > m ? v[p] : m;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long u = __shfl_xor_sync(kFull, m, o);
        m = u > m ? u : m;
    }
    if ((threadIdx.x & 31) == 0) atomicMax(out, m);
}

// ---- diagnostics: integer sums by atomics (order independent), fp64 sums per block in a fixed
// order and then over blocks in a fixed order (deterministic).
__global__ void __launch_bounds__(kThreads)
lp_diag_kernel(const int32_t *__restrict__ nsub, const double *__restrict__ lost,
               const int32_t *__restrict__ status, const double *__restrict__ chi,
               const double *__restrict__ eng, const double *__restrict__ tab, int nbins, long long np,
               double *__restrict__ partial, LpDiagDev *out)
{
    __shared__ double snum[kWarps], slost[kWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double *dE = tab + (nbins + 1);
    long long sum_ns = 0, capped = 0, outside = 0;
    int max_ns = 0;
    double lo = 0.0;
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < np; p += (long long)gridDim.x * blockDim.x) {
        int n = nsub[p];
        if (n < 0) { ++capped; n = -n; }
        sum_ns += n;
        max_ns = n > max_ns ? n : max_ns;
        if (status && status[p]) ++outside;
        if (lost) lo += lost[p];
    }
    double num = 0.0;
    const long long gw = (long long)blockIdx.x * kWarps + warp, nw = (long long)gridDim.x * kWarps;
    // four rows per trip (independent loads in flight); the sum order per lane is fixed by (gw, nw)
    for (long long r = gw; r < np; r += 4 * nw) {
        for (int i = lane; i < nbins; i += 32) {
            const double w = dE[i];
            double v[4], wk[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const long long rr = r + k * nw;
                v[k] = (rr < np) ? chi[rr * nbins + i] : 0.0;
                // moving grid: the particle's own bin widths
                wk[k] = (eng && rr < np) ? eng[rr * (nbins + 1) + i + 1] - eng[rr * (nbins + 1) + i] : w;
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) num = fma(v[k], wk[k], num);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sum_ns += __shfl_xor_sync(kFull, sum_ns, o);
        capped += __shfl_xor_sync(kFull, capped, o);
        outside += __shfl_xor_sync(kFull, outside, o);
        max_ns = max(max_ns, __shfl_xor_sync(kFull, max_ns, o));
        lo += __shfl_xor_sync(kFull, lo, o);
        num += __shfl_xor_sync(kFull, num, o);
    }
    if (lane == 0) {
        atomicAdd((unsigned long long *)&out->sum_substeps, (unsigned long long)sum_ns);
        atomicAdd((unsigned long long *)&out->n_capped, (unsigned long long)capped);
        atomicAdd((unsigned long long *)&out->n_outside, (unsigned long long)outside);
        atomicMax(&out->max_substeps, max_ns);
        snum[warp] = num;
        slost[warp] = lo;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < kWarps; ++w) { a += snum[w]; b += slost[w]; }
        partial[2 * blockIdx.x] = a;
        partial[2 * blockIdx.x + 1] = b;
    }
}

__global__ void lp_diag_final_kernel(const double *__restrict__ partial, int nblocks, LpDiagDev *out)
{
    double a = 0.0, b = 0.0;
    for (int i = 0; i < nblocks; ++i) { a += partial[2 * i]; b += partial[2 * i + 1]; }
    out->number = a;
    out->lost = b;
}

inline bool ok() { return cudaPeekAtLastError() == cudaSuccess; }

}  // namespace

size_t lp_sort_hist_elems(long long np) { return (size_t)256 * (size_t)blocks_for(np, kTile) + 256; }

// radix passes into b.idx_a / b.idx_b; enable (device flag, or NULL = always): see the counting sort
static int radix_passes(const uint64_t *id, long long np, int id_bits, int key_bits, const LpSortBufs &b,
                        const uint32_t *enable, uint32_t **perm_out, cudaStream_t s)
{
    int launches = 0;
    const int nblocks = blocks_for(np, kTile);
    const uint32_t *in = nullptr;       // identity
    uint32_t *bufs[2] = { b.idx_a, b.idx_b };
    int cur = 0;
    const int id_passes = (id_bits + 7) / 8, key_passes = (key_bits + 7) / 8;
    const int total = id_passes + key_passes;
    for (int pass = 0; pass < (total > 0 ? total : 1); ++pass) {
        const int use_key = pass >= id_passes ? 1 : 0;
        const int shift = 8 * (use_key ? pass - id_passes : pass);
        lp_radix_hist_kernel<<<nblocks, kThreads, 0, s>>>(in, id, b.key, np, use_key, shift, b.hist, nblocks, b.digit, enable);
        uint32_t *totals = b.hist + (size_t)256 * nblocks;
        lp_scan_rows_kernel<<<256, kThreads, 0, s>>>(b.hist, nblocks, totals, enable);
        lp_radix_scatter_kernel<<<nblocks, kThreads, 0, s>>>(in, id, b.key, np, use_key, shift, b.hist, totals, nblocks, bufs[cur],
                                                             b.digit, enable);
        launches += 3;
        in = bufs[cur];
        cur ^= 1;
    }
    *perm_out = const_cast<uint32_t *>(in);
    return launches;
}

int lp_launch_sort_perm(const LpGeom &g, const double *x, const double *y, const double *z, const uint64_t *id,
                        long long np, int id_bits, int key_bits, const LpSortBufs &b, uint32_t **perm_out,
                        cudaStream_t s)
{
    lp_key_kernel<<<blocks_for(np, kThreads), kThreads, 0, s>>>(g, x, y, z, np, b.key);
    const int launches = 1 + radix_passes(id, np, id_bits, key_bits, b, nullptr, perm_out, s);
    return ok() ? launches : -1;
}

size_t lp_sort_scan_tiles(long long ncell) { return (size_t)blocks_for(ncell, kScanTile); }

int lp_launch_sort_perm_counting(const LpGeom &g, const double *x, const double *y, const double *z,
                                 const uint64_t *id, long long np, int id_bits, int key_bits, const LpSortBufs &b,
                                 const LpCountBufs &cb, uint32_t **perm_out, cudaStream_t s)
{
    const long long ncell = (long long)g.nx * g.ny * g.nz;
    const int pblocks = blocks_for(np, kThreads), ntiles = blocks_for(ncell, kScanTile);
    if (cudaMemsetAsync(cb.cnt, 0, (size_t)(ncell + 1) * 4, s) != cudaSuccess) return -1;
    if (cudaMemsetAsync(cb.overflow, 0, 4, s) != cudaSuccess) return -1;
    uint32_t *rank0 = b.idx_a, *perm = b.idx_b;
    lp_cell_count_kernel<<<pblocks, kThreads, 0, s>>>(g, x, y, z, np, b.key, cb.cnt, rank0);
    lp_scan_tile_sums_kernel<<<ntiles, kThreads, 0, s>>>(cb.cnt, ncell, cb.tile_sum);
    lp_scan_tile_offsets_kernel<<<1, kThreads, 0, s>>>(cb.tile_sum, ntiles);
    lp_scan_tiles_kernel<<<ntiles, kThreads, 0, s>>>(cb.cnt, ncell, cb.tile_sum);
    lp_cell_place_kernel<<<pblocks, kThreads, 0, s>>>(b.key, rank0, cb.cnt, id, np, cb.seg_id);
    lp_cell_rank_kernel<<<pblocks, kThreads, 0, s>>>(b.key, cb.cnt, id, cb.seg_id, np, perm, cb.overflow);
    int launches = 6;
    // fallback, gated on *overflow: the radix sort of the same keys, its result copied over perm
    uint32_t *rperm = nullptr;
    launches += radix_passes(id, np, id_bits, key_bits, b, cb.overflow, &rperm, s);
    if (rperm != perm) {
        lp_copy_if_kernel<<<blocks_for(np, kThreads * 8), kThreads, 0, s>>>(rperm, perm, np, cb.overflow);
        ++launches;
    }
    *perm_out = perm;
    return ok() ? launches : -1;
}

int lp_launch_permute_f64(const uint32_t *perm, const double *src, double *dst, long long np, cudaStream_t s)
{
    lp_permute_f64_kernel<<<blocks_for(np, kThreads), kThreads, 0, s>>>(perm, src, dst, np);
    return ok() ? 1 : -1;
}

int lp_launch_permute_u64(const uint32_t *perm, const uint64_t *src, uint64_t *dst, long long np, cudaStream_t s)
{
    lp_permute_u64_kernel<<<blocks_for(np, kThreads), kThreads, 0, s>>>(perm, src, dst, np);
    return ok() ? 1 : -1;
}

int lp_launch_permute_rows(const uint32_t *perm, const double *src, double *dst, long long np, int nbins,
                           cudaStream_t s)
{
    const int lanes = nbins / 2 < 32 ? nbins / 2 : 32;
    const long long warps = (np + (32 / lanes) - 1) / (32 / lanes);
    long long blocks = (warps + kWarps - 1) / kWarps;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (blocks < 1) blocks = 1;
    lp_permute_rows_kernel<<<(int)blocks, kThreads, 0, s>>>(perm, src, dst, np, nbins);
    return ok() ? 1 : -1;
}

int lp_launch_max_u64(const uint64_t *v, long long np, unsigned long long *out, cudaStream_t s)
{
    int blocks = blocks_for(np, kThreads * 8);
    if (blocks > 1024) blocks = 1024;
    lp_max_u64_kernel<<<blocks, kThreads, 0, s>>>(v, np, out);
    return ok() ? 1 : -1;
}

int lp_launch_diag(const int32_t *nsub, const double *lost, const int32_t *status, const double *chi,
                   const double *eng, const double *tab, int nbins, long long np, double *partial, LpDiagDev *out,
                   cudaStream_t s)
{
    const int blocks = 296;      // (the scratch `partial` holds 2 x 296 doubles)
    lp_diag_kernel<<<blocks, kThreads, 0, s>>>(nsub, lost, status, chi, eng, tab, nbins, np, partial, out);
    lp_diag_final_kernel<<<1, 1, 0, s>>>(partial, blocks, out);
    return ok() ? 2 : -1;
}
