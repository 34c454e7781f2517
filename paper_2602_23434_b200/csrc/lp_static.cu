// lp_static.cu -- lp_number_static: the particle number  sum_p sum_i chi[p][i] dE[i]  of a set of spectra,
// computed without allocating anything, anywhere.
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Who this is for.  Every other reduction of this library goes through a context: lp_create uploads a bin
// table with cudaMalloc, and lp_get_diag keeps its per-block partial sums in the caller's workspace, which
// somebody had to allocate too (several GB at workload size, because it is sized for the whole step).  Some
// users of an LP module have no way to do either at the moment they want the number:
//   * an in-situ conservation monitor hooked into a host code (PLUTO itself, or an OpenACC / MPI driver around
//     it) that handed all device memory to its own arena at start-up: there is nothing left to cudaMalloc
//     from, and the arena is not ours to carve;
//   * a callback that runs while other streams are busy: cudaMalloc and cudaFree synchronise the whole device,
//     so a "cheap" diagnostic would stall the step it is watching;
//   * code between cudaStreamBeginCapture and cudaStreamEndCapture of somebody else's graph, where the
//     allocating runtime calls are simply illegal.
// For them the scratch of the reduction (one partial sum per tile of rows) lives in a file-scope __device__
// array below: 64 KiB that every GPU which loads liblp_b200.so holds from module load until the process exits,
// whether or not this call is ever made.  That fixed size is where the row limit comes from.
//
// The kernel is a variant of lp_diag_kernel (lp_sort.cu), the `number` part only, with one change that the
// fixed scratch invites: the tiling depends on the row count alone (2048 rows per block, one partial per
// block, partials added in ascending order), not on the launch grid, so the result is the same bit pattern on
// any GPU and in any process.  lp_get_diag sums in another order; the two agree to rounding (a few ulp of the
// sum), which is what tests/test_zz_no_alloc.py checks.
#include <cstdio>
#include <mutex>
#include <cuda_runtime.h>
#include "../../include/lp.h"

namespace {

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kRowsPerTile = 2048;
constexpr int kMaxTiles = (int)(LP_NUMBER_STATIC_MAX_NP / kRowsPerTile);      // 8192
constexpr int kMaxDevices = 64;
constexpr unsigned kFull = 0xffffffffu;

static_assert((long long)kMaxTiles * kRowsPerTile == LP_NUMBER_STATIC_MAX_NP, "row limit is a whole number of tiles");

// The scratch.  In device code this name is the array; in host code it is only a handle for
// cudaGetSymbolAddress -- never a pointer to hand to a kernel (see device_scratch below).
static __device__ __align__(256) double lp_static_partial[kMaxTiles];         // 8192 x 8 B = 64 KiB per GPU

// partial[b] = sum over rows [b*2048, min(np, (b+1)*2048)) of sum_i chi[row][i] * dE[i]; the order of the
// additions is fixed by (row count, nbins) alone.
__global__ void __launch_bounds__(kThreads)
lp_number_tile_kernel(const double *__restrict__ chi, const double *__restrict__ dE, int nbins, long long np,
                      double *__restrict__ partial)
{
    __shared__ double swarp[kWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long r0 = (long long)blockIdx.x * kRowsPerTile;
    const long long r1 = (r0 + kRowsPerTile < np) ? r0 + kRowsPerTile : np;
    double num = 0.0;
    // a warp per row, four rows of a warp in flight per trip
    for (long long r = r0 + warp; r < r1; r += 4 * kWarps) {
        for (int i = lane; i < nbins; i += 32) {
            const double w = __ldg(dE + i);
            double v[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const long long rr = r + (long long)k * kWarps;
                v[k] = (rr < r1) ? __ldcs(chi + rr * nbins + i) : 0.0;
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) num = fma(v[k], w, num);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) num += __shfl_xor_sync(kFull, num, o);
    if (lane == 0) swarp[warp] = num;
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0;
        for (int w = 0; w < kWarps; ++w) a += swarp[w];
        partial[blockIdx.x] = a;            // every slot [0, ntiles) is overwritten before the final kernel reads it
    }
}

// one block: thread t adds partial[t], partial[t + 256], ... in ascending order, then a fixed tree over the threads
__global__ void __launch_bounds__(kThreads)
lp_number_final_kernel(const double *__restrict__ partial, int ntiles, double *__restrict__ number)
{
    __shared__ double s[kThreads];
    double a = 0.0;
    for (int i = threadIdx.x; i < ntiles; i += kThreads) a += partial[i];
    s[threadIdx.x] = a;
    __syncthreads();
    for (int h = kThreads / 2; h > 0; h >>= 1) {
        if ((int)threadIdx.x < h) s[threadIdx.x] += s[threadIdx.x + h];
        __syncthreads();
    }
    if (threadIdx.x == 0) *number = s[0];
}

// Device address of lp_static_partial on `device` (which must be current), looked up once per device.
std::mutex g_lock;
double *g_scratch[kMaxDevices];       // zero-initialised: not looked up yet

cudaError_t device_scratch(int device, double **out)
{
    std::lock_guard<std::mutex> hold(g_lock);
    if (!g_scratch[device]) {
        void *p = nullptr;
        // Loads this module's image on the device if nothing of the library ran there yet, which is
        // driver-side work that does not belong inside a stream capture: hence "first call per device
        // before any capture" in lp.h.
        const cudaError_t e = cudaGetSymbolAddress(&p, lp_static_partial);
        if (e != cudaSuccess) return e;
        g_scratch[device] = static_cast<double *>(p);
    }
    *out = g_scratch[device];
    return cudaSuccess;
}

lp_status say(lp_status st, char *err, size_t err_len, const char *fmt, long long a = 0, long long b = 0)
{
    if (err && err_len) std::snprintf(err, err_len, fmt, a, b);
    return st;
}

lp_status say_cuda(cudaError_t e, const char *what, char *err, size_t err_len)
{
    if (err && err_len) std::snprintf(err, err_len, "%s: %s", what, cudaGetErrorString(e));
    return LP_ERR_CUDA;
}

}  // namespace

extern "C" lp_status lp_number_static(int device, const double *chi, const double *widths, int32_t nbins, int64_t np,
                                      double *number, void *stream, char *err, size_t err_len)
{
    if (err && err_len) err[0] = '\0';
    if (device < 0 || device >= kMaxDevices)
        return say(LP_ERR_INVALID_ARG, err, err_len, "device %lld outside [0, %lld)", device, kMaxDevices);
    if (np < 0) return say(LP_ERR_INVALID_ARG, err, err_len, "np = %lld is negative", np);
    if (nbins < 1 || nbins > LP_NUMBER_STATIC_MAX_NBINS)
        return say(LP_ERR_UNSUPPORTED, err, err_len, "nbins = %lld outside [1, %lld]", nbins, LP_NUMBER_STATIC_MAX_NBINS);
    if (np > LP_NUMBER_STATIC_MAX_NP)
        return say(LP_ERR_UNSUPPORTED, err, err_len,
                   "np = %lld rows exceed the %lld the static scratch of lp_number_static holds partial sums for "
                   "(call it on slices, or use lp_get_diag with a workspace)", np, LP_NUMBER_STATIC_MAX_NP);
    if (!number || !widths || (np > 0 && !chi))
        return say(LP_ERR_INVALID_ARG, err, err_len, "chi, widths or number is NULL");

    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e != cudaSuccess) return say_cuda(e, "cudaGetDevice", err, err_len);
    if (prev != device && (e = cudaSetDevice(device)) != cudaSuccess) return say_cuda(e, "cudaSetDevice", err, err_len);

    lp_status st = LP_OK;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    double *scratch = nullptr;
    if ((e = device_scratch(device, &scratch)) != cudaSuccess) {
        st = say_cuda(e, "cudaGetSymbolAddress(lp_static_partial)", err, err_len);
    } else if (np == 0) {
        if ((e = cudaMemsetAsync(number, 0, sizeof(double), s)) != cudaSuccess) st = say_cuda(e, "cudaMemsetAsync", err, err_len);
    } else {
        const int ntiles = (int)((np + kRowsPerTile - 1) / kRowsPerTile);
        lp_number_tile_kernel<<<ntiles, kThreads, 0, s>>>(chi, widths, nbins, np, scratch);
        lp_number_final_kernel<<<1, kThreads, 0, s>>>(scratch, ntiles, number);
        if ((e = cudaPeekAtLastError()) != cudaSuccess) st = say_cuda(e, "lp_number_static launch", err, err_len);
    }
    if (prev != device) cudaSetDevice(prev);
    return st;
}
