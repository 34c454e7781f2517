// lp_internal.h -- host-side declarations shared by the translation units of liblp_b200.so.
// Product code (CUDA path).  Shares nothing with oracle/.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/lp.h"

// Grid geometry handed to kernels by value (fits in kernel-parameter constant bank).
struct LpGeom {
    int nx, ny, nz;
    int per[3];
    double xlo[3], xhi[3];
    double inv_dx[3];        // n / (xhi - xlo), computed on the host in fp64
    double len[3];           // xhi - xlo
};

// Per-cell records built by lp_set_fields, two 32-byte halves per cell,
//   A = (vx, vy, vz, rho)    B = (bx, by, bz, 0),
// half A of cell c at recA[stride * c], half B at recB[stride * c], in one of two layouts chosen at lp_create:
//  * stride 2, recB = recA + 1: one 64-byte record per cell.  A 64-byte record is one DRAM access whatever
//    its alignment, so a particle with no neighbour in its cells fetches 8 x 64 bytes, all but 8 of them used,
//    where separate 32-byte arrays fetch 1.5 x that (DRAM moves 64 bytes at a time).  The layout for sparse
//    particle sets (fewer particles than cells): workload 5 gains 10-22 %, workload 3 2 %.
//  * stride 1, recB = recA + cells: two arrays.  With a particle or more in every cell the A halves are read
//    three times per step by neighbouring particles and four of them share an L1 line; workload 4 is 3 %
//    faster this way (measured, profiles/r02_gather_layout.md).
struct LpCells {
    const double4 *recA;
    const double4 *recB;
    unsigned stride;
};

// Bins at which the outflow rate (max(w_{i+1},0) - min(w_i,0))/dE_i can be the maximum over the
// row for some (a, c_r >= 0): both clamped terms are linear in (a, c_r), so the maximum over bins is
// attained at a vertex of the convex hull of their coefficient points; lp_create finds those
// vertices once per bin table (on a log grid: the two end bins plus rounding-noise neighbours).
// n < 0: table degenerate, scan every bin.
constexpr int kLpMaxCand = 24;
struct LpLamCand {
    int n;
    int bin[kLpMaxCand];
    double el[kLpMaxCand], er[kLpMaxCand], rde[kLpMaxCand];   // E_i, E_{i+1}, 1/dE_i of those bins
    double margin;      // relative bound on how far the maximum over all bins can exceed that of bins 0, N_b-1
};

struct LpSpectralArgs {
    LpGeom g;
    LpLamCand cand;
    LpCells cells;
    double *x, *y, *z;           // staged: x^{n+1} (read only).  fused: x^{n+1} out
    const double *xin, *yin, *zin;   // positions read (== x, y, z unless the step re-sorts: the other buffer set)
    // Re-sort folded into the fused step (lp_step on a sort step, ping-pong buffers): particle p of the new
    // order is the particle stored at index perm[p] of xin, yin, zin, id_in and chi_in; everything is written
    // at index p of the other buffer set (x, y, z, id_out, chi_out), so the row permute costs no pass of its
    // own.  perm == NULL: identity (no re-sort), id_in / id_out unused.
    const uint32_t *perm;
    const uint64_t *id_in;
    uint64_t *id_out;
    const double *rho_old;       // staged: from push stage 0.  fused: unused
    int32_t *status;             // fused: outside-box flags [np]
    const double *chi_in;        // [np][nbins]  (may differ from chi_out after a re-sort)
    double *chi_out;             // [np][nbins]
    const double *tab;           // device bin table: E[nb+1] | dE[nb] | rdE[nb]
    int32_t *nsub_ws;            // [np] always written (workspace)
    int32_t *nsub_user;          // [np] or NULL
    double *lost_ws;             // [np] always written when DIAG
    double *lost_user;           // [np] or NULL
    long long np;
    double dt, kappa, u_rad, cfl_e;
    int max_substeps;
};

struct LpPushArgs {
    LpGeom g;
    LpCells cells;
    double *x, *y, *z;           // bound positions (x^n in, x^{n+1} out at stage 1)
    double *k1;                  // [3][np]
    double *xs;                  // [3][np]  predictor positions
    double *rho_old;             // [np]
    int32_t *status;             // [np]
    long long np;
    double dt;
};

// ---- launchers (each returns the number of kernels it enqueued, or -1 with cudaGetLastError set)
int lp_launch_repack(const double *const f[7], double4 *recA, double4 *recB, unsigned stride, long long ncell,
                     cudaStream_t s);
int lp_launch_interpolate(const LpGeom &g, const LpCells &c, const double *x, const double *y,
                          const double *z, long long np, double *out7, uint32_t *key, cudaStream_t s);
int lp_launch_interpolate_tiled(const LpGeom &g, const LpCells &c, const double *x, const double *y,
                                const double *z, long long np, double *out7, bool *configured, cudaStream_t s);
int lp_launch_push0(const LpPushArgs &a, cudaStream_t s);
int lp_launch_push1(const LpPushArgs &a, cudaStream_t s);
int lp_launch_push_rk3(const LpPushArgs &a, int stage, cudaStream_t s);     // stage 0, 1, 2 (x0 kept in a.xs)
// fused = true: the kernel also does both push stages (a5, a6) in its per-particle phase (frozen fields)
// blocks_cache: int[6] owned by the context, [diag][mode: staged, fused, fused + re-sort] resident blocks per SM
// (0 = variant not set up yet)
int lp_launch_spectral(const LpSpectralArgs &a, int nbins, bool diag, bool fused, int sm_count, int *blocks_cache,
                       cudaStream_t s);

// shock-crossing update of the flagged rows (lp_shock.cu); r [np] device, r <= 1 = untouched
// eng != NULL: every row on its own edges eng[p][0..nbins] (moving energy grid) instead of the table's
int lp_launch_shock(const double *tab, const double *eng, const double *r, double q_r, double *chi, long long np,
                    int nbins, int sm_count, cudaStream_t s);

// deletion with hole filling (lp_compact.cu); counts = 2 x u64 on the device: N_del, number of holes
size_t lp_compact_block_elems(long long np);
int lp_launch_compact(const int32_t *flag, long long np, int nbins, uint32_t *blk, uint32_t *rank, uint32_t *hole,
                      uint32_t *filler, unsigned long long *counts, double *x, double *y, double *z, uint64_t *id,
                      double *chi, double *eng /*or NULL*/, int sm_count, cudaStream_t s);

// particle exchange (lp_migrate.cu); counts = 2 x u64 on the device: n_left, n_right
size_t lp_migrate_block_elems(long long np);
int lp_launch_migrate_count(const double *pos, long long np, double lo, double hi, double len, int periodic,
                            uint32_t *dest, unsigned long long *blk, unsigned long long *counts, uint32_t *hole,
                            uint32_t *leaver, cudaStream_t s);
int lp_launch_migrate_pack(long long n_left, long long n_right, const uint32_t *leaver,
                           const double *x, const double *y, const double *z, const uint64_t *id, const double *chi,
                           const double *eng /*or NULL*/, int nbins, void *buf_left, void *buf_right, int sm_count,
                           cudaStream_t s);
int lp_launch_migrate_unpack(const void *in_left, long long n_in_left, const void *in_right, long long n_in_right,
                             const uint32_t *hole, long long nholes, long long np, double *x, double *y, double *z,
                             uint64_t *id, double *chi, double *eng /*or NULL*/, int nbins, int32_t *flag_rest,
                             int sm_count, cudaStream_t s);

// sort: fills perm[n] = source index of the n-th particle in (key, id) order.
struct LpSortBufs {
    uint32_t *key;       // [np]
    uint32_t *idx_a;     // [np]
    uint32_t *idx_b;     // [np]
    uint32_t *hist;      // [256 * nblocks]
    size_t hist_elems;
    uint8_t *digit;      // [np] digit of every element of the current pass (hist kernel -> scatter kernel)
};
size_t lp_sort_hist_elems(long long np);
int lp_launch_sort_perm(const LpGeom &g, const double *x, const double *y, const double *z,
                        const uint64_t *id, long long np, int id_bits, int key_bits,
                        const LpSortBufs &b, uint32_t **perm_out, cudaStream_t s);
// Counting sort by cell (lp_sort.cu): one counter per cell plus rank counting inside the cells; falls back to
// the radix passes on the device when a cell holds more than 64 particles.  id_bits: as for the radix sort
// (64 when not measured).
struct LpCountBufs {
    uint32_t *cnt;       // [ncell + 1]  counters, then exclusive offsets
    uint32_t *tile_sum;  // [lp_sort_scan_tiles(ncell)]
    uint64_t *seg_id;    // [np]  ids grouped by cell (scratch: the id array of the other buffer set)
    uint32_t *overflow;  // [1]
};
size_t lp_sort_scan_tiles(long long ncell);
int lp_launch_sort_perm_counting(const LpGeom &g, const double *x, const double *y, const double *z,
                                 const uint64_t *id, long long np, int id_bits, int key_bits, const LpSortBufs &b,
                                 const LpCountBufs &cb, uint32_t **perm_out, cudaStream_t s);
int lp_launch_permute_f64(const uint32_t *perm, const double *src, double *dst, long long np, cudaStream_t s);
int lp_launch_permute_u64(const uint32_t *perm, const uint64_t *src, uint64_t *dst, long long np, cudaStream_t s);
int lp_launch_permute_rows(const uint32_t *perm, const double *src, double *dst, long long np,
                           int nbins, cudaStream_t s);
int lp_launch_max_u64(const uint64_t *v, long long np, unsigned long long *out, cudaStream_t s);

// moving energy grid (lp_moving.cu)
// fused: the kernel also does both push stages (x^n read, x^{n+1} and status written), rho_old unused.
// io.perm != NULL (fused only): the step re-sorts -- everything is read at perm[p] of the *_in arrays and written
// at p of the others.
struct LpMovingIO {
    const double *xin, *yin, *zin, *eng_in, *chi_in;
    double *x, *y, *z, *eng, *chi;
    const uint32_t *perm;
    const uint64_t *id_in;
    uint64_t *id_out;
};
int lp_launch_moving(const LpGeom &g, const LpCells &cells, const LpMovingIO &io, const double *rho_old, int32_t *status,
                     bool fused, int32_t *nsub_ws, int32_t *nsub_user, long long np, int nbins, double dt, double kappa,
                     double u_rad, int sm_count, cudaStream_t s);
int lp_launch_moving_init(const double *tab, int nbins, double *eng, long long first, long long count, cudaStream_t s);
int lp_launch_permute_rows8(const uint32_t *perm, const double *src, double *dst, long long np, int len, cudaStream_t s);

// diagnostics reduction
struct LpDiagDev {
    long long sum_substeps;
    long long n_capped;
    long long n_outside;
    int max_substeps;
    int pad;
    double number;
    double lost;
};
int lp_launch_diag(const int32_t *nsub, const double *lost, const int32_t *status, const double *chi,
                   const double *eng /*[np][nbins+1] per-particle edges, or NULL: the table's widths*/, const double *tab, int nbins, long long np, double *partial /*scratch*/,
                   LpDiagDev *out, cudaStream_t s);
