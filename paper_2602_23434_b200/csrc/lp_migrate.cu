// lp_migrate.cu -- exchange of the particles that crossed a rank interface (readings M1-M3
// of DESIGN.md section 3), the kernels of one rank and one direction:
//   count   (step 1)  destination of every particle (0 stay, 1 left, 2 right) and the two totals
//   list    (step 1)  the leavers in ascending index order: holes[], left list, right list -- their ranks
//                     come from ONE exclusive prefix sum over a packed (left, right) counter pair
//   pack    (step 4)  a warp per leaver copies x, y, z, id and the chi row into the neighbour's send buffer
//   unpack  (step 8)  a warp per arrival: k-th arrival (left buffer first) into the k-th hole, or behind the
//                     last particle when the holes are used up; holes that stay open are flagged for the
//                     compaction of lp_compact.cu
// A send buffer for n particles is laid out as arrays: x[n] | y[n] | z[n] | id[n] | chi[n][nbins]
// [| eng[n][nbins+1] when the particles carry an energy grid]  (n * lp_migrate_record_bytes bytes, 16-byte
// aligned base), so both sides of the copy are coalesced and the buffer is what one NCCL send / NVLink peer copy
// moves.  sm_100a.
#include "lp_internal.h"

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kItems = 16;
constexpr int kTile = kThreads * kItems;

inline int blocks_for(long long n, int per) { long long b = (n + per - 1) / per; return (int)(b < 1 ? 1 : b); }

// Reading M1.  Every operation is one rounded fp64 operation in the order the oracle writes them.
__device__ __forceinline__ uint32_t lp_mig_dest(double x, double lo, double hi, double L, int periodic)
{
    if (x >= lo && x < hi) return 0u;
    if (x < lo) {
        if (periodic) {
            const double left = __dsub_rn(lo, x), right = __dsub_rn(__dadd_rn(x, L), hi);
            if (right >= 0.0 && right < left) return 2u;
        }
        return 1u;
    }
    if (periodic) {
        const double right = __dsub_rn(x, hi), left = __dsub_rn(lo, __dsub_rn(x, L));
        if (left >= 0.0 && left < right) return 1u;
    }
    return 2u;
}

// packed pair of counters: left in the low, right in the high 32 bits (np < 2^32)
__device__ __forceinline__ unsigned long long lp_pair(uint32_t d)
{
    return d == 1u ? 1ull : (d == 2u ? (1ull << 32) : 0ull);
}

__device__ __forceinline__ unsigned long long block_excl_scan64(unsigned long long v, unsigned long long *total)
{
    __shared__ unsigned long long wsum[kWarps];
    __shared__ unsigned long long tot;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long u = __shfl_up_sync(kFull, inc, o);
        if (lane >= o) inc += u;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    unsigned long long wbase = 0;
    for (int w = 0; w < warp; ++w) wbase += wsum[w];
    if (threadIdx.x == kThreads - 1) tot = wbase + inc;
    __syncthreads();
    *total = tot;
    const unsigned long long r = wbase + inc - v;
    __syncthreads();
    return r;
}

// step 1a: destinations of a tile (thread t owns items t*kItems .., so ranks follow the index order)
__global__ void __launch_bounds__(kThreads)
lp_mig_count_kernel(const double *__restrict__ pos, long long np, double lo, double hi, double L, int periodic,
                    uint32_t *__restrict__ dest, unsigned long long *__restrict__ blk)
{
    const long long i0 = (long long)blockIdx.x * kTile + (long long)threadIdx.x * kItems;
    unsigned long long c = 0;
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        if (i0 + k < np) {
            const uint32_t d = lp_mig_dest(pos[i0 + k], lo, hi, L, periodic);
            dest[i0 + k] = d;
            c += lp_pair(d);
        }
    }
    unsigned long long total;
    block_excl_scan64(c, &total);
    if (threadIdx.x == 0) blk[blockIdx.x] = total;
}

// step 1b: exclusive scan of the block totals (one block); counts[0] = n_left, counts[1] = n_right
__global__ void __launch_bounds__(kThreads)
lp_mig_scan_kernel(unsigned long long *__restrict__ blk, int nblocks, unsigned long long *__restrict__ counts)
{
    unsigned long long carry = 0;
    for (int b0 = 0; b0 < nblocks; b0 += kThreads) {
        const int i = b0 + threadIdx.x;
        const unsigned long long v = i < nblocks ? blk[i] : 0ull;
        unsigned long long total;
        const unsigned long long ex = block_excl_scan64(v, &total);
        if (i < nblocks) blk[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0) {
        counts[0] = carry & 0xffffffffull;
        counts[1] = carry >> 32;
    }
}

// step 1c: the ordered lists.  hole[k] = k-th leaver; leaver[0 .. n_left) those going left, leaver[n_left ..)
// those going right, each ascending.
__global__ void __launch_bounds__(kThreads)
lp_mig_list_kernel(const uint32_t *__restrict__ dest, long long np, const unsigned long long *__restrict__ blk,
                   const unsigned long long *__restrict__ counts, uint32_t *__restrict__ hole,
                   uint32_t *__restrict__ leaver)
{
    const long long i0 = (long long)blockIdx.x * kTile + (long long)threadIdx.x * kItems;
    uint32_t d[kItems];
    unsigned long long c = 0;
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        d[k] = i0 + k < np ? dest[i0 + k] : 0u;
        c += lp_pair(d[k]);
    }
    unsigned long long total;
    unsigned long long run = blk[blockIdx.x] + block_excl_scan64(c, &total);
    const uint32_t nl = (uint32_t)counts[0];
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        if (d[k]) {
            const uint32_t rl = (uint32_t)(run & 0xffffffffull), rr = (uint32_t)(run >> 32);
            hole[rl + rr] = (uint32_t)(i0 + k);
            leaver[d[k] == 1u ? rl : nl + rr] = (uint32_t)(i0 + k);
            run += lp_pair(d[k]);
        }
    }
}

struct LpMigBuf {           // one send / receive buffer, as arrays
    double *x, *y, *z;
    uint64_t *id;
    double *chi;
    double *eng;            // [n][nbins + 1] behind chi when the particles carry an energy grid
};

__device__ __forceinline__ LpMigBuf lp_mig_view(void *base, unsigned long long n, int nbins)
{
    LpMigBuf b;
    b.x = static_cast<double *>(base);
    b.y = b.x + n;
    b.z = b.y + n;
    b.id = reinterpret_cast<uint64_t *>(b.z + n);
    b.chi = reinterpret_cast<double *>(b.id + n);
    b.eng = b.chi + n * (unsigned long long)nbins;
    return b;
}

// step 4: a warp per leaver
__global__ void __launch_bounds__(kThreads)
lp_mig_pack_kernel(unsigned long long nl, unsigned long long nr, const uint32_t *__restrict__ leaver,
                   const double *__restrict__ x, const double *__restrict__ y, const double *__restrict__ z,
                   const uint64_t *__restrict__ id, const double *__restrict__ chi, const double *__restrict__ eng,
                   int nbins, void *buf_left, void *buf_right)
{
    // (nl, nr by value: the host holds them since lp_migrate_count synchronised for them, and the device copy sits in
    // scratch that lp_get_diag may overwrite between count and pack)
    const LpMigBuf L = lp_mig_view(buf_left, nl, nbins), R = lp_mig_view(buf_right, nr, nbins);
    const int lane = threadIdx.x & 31;
    const long long gw = ((long long)blockIdx.x * kThreads + threadIdx.x) >> 5;
    const long long nw = ((long long)gridDim.x * kThreads) >> 5;
    for (long long k = gw; k < (long long)(nl + nr); k += nw) {
        const bool right = k >= (long long)nl;
        const LpMigBuf &B = right ? R : L;
        const long long d = right ? k - (long long)nl : k;
        const long long s = leaver[k];
        if (lane == 0) { B.x[d] = x[s]; B.y[d] = y[s]; B.z[d] = z[s]; B.id[d] = id[s]; }
        const double2 *src = reinterpret_cast<const double2 *>(chi + s * nbins);
        double2 *dst = reinterpret_cast<double2 *>(B.chi + d * nbins);
        for (int i = lane; i < nbins / 2; i += 32) dst[i] = src[i];
        if (eng)
            for (int i = lane; i <= nbins; i += 32) B.eng[d * (nbins + 1) + i] = eng[s * (nbins + 1) + i];
    }
}

// step 8: a warp per arrival
__global__ void __launch_bounds__(kThreads)
lp_mig_unpack_kernel(const void *in_left, long long n_in_left, const void *in_right, long long n_in_right,
                     const uint32_t *__restrict__ hole, long long nholes, long long np,
                     double *__restrict__ x, double *__restrict__ y, double *__restrict__ z,
                     uint64_t *__restrict__ id, double *__restrict__ chi, double *__restrict__ eng, int nbins)
{
    const LpMigBuf L = lp_mig_view(const_cast<void *>(in_left), (unsigned long long)n_in_left, nbins);
    const LpMigBuf R = lp_mig_view(const_cast<void *>(in_right), (unsigned long long)n_in_right, nbins);
    const int lane = threadIdx.x & 31;
    const long long gw = ((long long)blockIdx.x * kThreads + threadIdx.x) >> 5;
    const long long nw = ((long long)gridDim.x * kThreads) >> 5;
    for (long long k = gw; k < n_in_left + n_in_right; k += nw) {
        const bool right = k >= n_in_left;
        const LpMigBuf &B = right ? R : L;
        const long long s = right ? k - n_in_left : k;
        const long long d = k < nholes ? (long long)hole[k] : np + (k - nholes);
        if (lane == 0) { x[d] = B.x[s]; y[d] = B.y[s]; z[d] = B.z[s]; id[d] = B.id[s]; }
        const double2 *src = reinterpret_cast<const double2 *>(B.chi + s * nbins);
        double2 *dst = reinterpret_cast<double2 *>(chi + d * nbins);
        for (int i = lane; i < nbins / 2; i += 32) dst[i] = src[i];
        if (eng)
            for (int i = lane; i <= nbins; i += 32) eng[d * (nbins + 1) + i] = B.eng[s * (nbins + 1) + i];
    }
}

// holes that no arrival filled: flag them for the compaction
__global__ void __launch_bounds__(kThreads)
lp_mig_flag_rest_kernel(const uint32_t *__restrict__ hole, long long first, long long nholes, int32_t *__restrict__ flag)
{
    const long long k = first + (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < nholes) flag[hole[k]] = 1;
}

inline bool ok() { return cudaPeekAtLastError() == cudaSuccess; }

}  // namespace

size_t lp_migrate_block_elems(long long np) { return (size_t)blocks_for(np, kTile) + 1; }

int lp_launch_migrate_count(const double *pos, long long np, double lo, double hi, double len, int periodic,
                            uint32_t *dest, unsigned long long *blk, unsigned long long *counts, uint32_t *hole,
                            uint32_t *leaver, cudaStream_t s)
{
    const int nblocks = blocks_for(np, kTile);
    lp_mig_count_kernel<<<nblocks, kThreads, 0, s>>>(pos, np, lo, hi, len, periodic, dest, blk);
    lp_mig_scan_kernel<<<1, kThreads, 0, s>>>(blk, nblocks, counts);
    lp_mig_list_kernel<<<nblocks, kThreads, 0, s>>>(dest, np, blk, counts, hole, leaver);
    return ok() ? 3 : -1;
}

int lp_launch_migrate_pack(long long n_left, long long n_right, const uint32_t *leaver,
                           const double *x, const double *y, const double *z, const uint64_t *id, const double *chi,
                           const double *eng, int nbins, void *buf_left, void *buf_right, int sm_count, cudaStream_t s)
{
    long long blocks = (n_left + n_right + kWarps - 1) / kWarps;
    const long long cap = (long long)sm_count * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    lp_mig_pack_kernel<<<(int)blocks, kThreads, 0, s>>>((unsigned long long)n_left, (unsigned long long)n_right, leaver, x, y, z, id, chi, eng, nbins, buf_left, buf_right);
    return ok() ? 1 : -1;
}

int lp_launch_migrate_unpack(const void *in_left, long long n_in_left, const void *in_right, long long n_in_right,
                             const uint32_t *hole, long long nholes, long long np, double *x, double *y, double *z,
                             uint64_t *id, double *chi, double *eng, int nbins, int32_t *flag_rest, int sm_count,
                             cudaStream_t s)
{
    int launches = 0;
    const long long nin = n_in_left + n_in_right;
    if (nin > 0) {
        long long blocks = (nin + kWarps - 1) / kWarps;
        const long long cap = (long long)sm_count * 8;
        if (blocks > cap) blocks = cap;
        lp_mig_unpack_kernel<<<(int)blocks, kThreads, 0, s>>>(in_left, n_in_left, in_right, n_in_right, hole, nholes,
                                                             np, x, y, z, id, chi, eng, nbins);
        ++launches;
    }
    if (nin < nholes && flag_rest) {
        lp_mig_flag_rest_kernel<<<blocks_for(nholes - nin, kThreads), kThreads, 0, s>>>(hole, nin, nholes, flag_rest);
        ++launches;
    }
    return ok() ? launches : -1;
}
