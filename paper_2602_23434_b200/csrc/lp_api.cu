// lp_api.cu -- the C ABI of include/lp.h: context, validation, workspace layout, launch order.
// Host code only; every step of the path runs in the kernels of lp_particles.cu, lp_spectral.cu
// and lp_sort.cu.  No CPU fallback exists.
#include <algorithm>
#include <utility>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "lp_internal.h"

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

struct Layout {
    size_t rec, k1, xs, rho_old, nsub, lost, status, key, idx_a, idx_b, hist, alt_id, pos_alt, chi_alt,
        partial, diag, maxid, cellcnt, tile_sum, total;
    size_t hist_elems;
    bool counting;          // sort by one counter per cell (else radix passes only)
};

Layout make_layout(const lp_config &c)
{
    Layout L{};
    const size_t ncell = (size_t)c.nx * c.ny * c.nz;
    const size_t np = (size_t)c.np;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    L.rec = take(ncell * 64);
    L.k1 = take(np * 24);
    L.xs = take(np * 24);
    L.rho_old = take(np * 8);
    L.nsub = take(np * 4);
    L.lost = take(np * 8);
    L.status = take(np * 4);
    L.key = take(np * 4);
    L.idx_a = take(np * 4);
    L.idx_b = take(np * 4);
    L.hist_elems = lp_sort_hist_elems(c.np);
    L.hist = take(L.hist_elems * 4);
    L.alt_id = take(np * 8);
    L.pos_alt = take(np * 24);
    L.chi_alt = take(np * (size_t)c.nbins * 8);
    L.partial = take(2 * 296 * 8);
    L.diag = take(sizeof(LpDiagDev));
    L.maxid = take(16);                  // largest id | overflow flag of the counting sort
    // Counting sort by cell: 4 bytes per cell.  Worth it unless the grid dwarfs the particle set (then the
    // O(cells) scan costs more than the radix passes over the particles it replaces).
    L.counting = ncell <= 64 * (np > 0 ? np : 1);
    L.cellcnt = take(L.counting ? (ncell + 1) * 4 : 0);
    L.tile_sum = take(L.counting ? lp_sort_scan_tiles((long long)ncell) * 4 : 0);
    L.total = off;
    return L;
}

// Bins that can carry the maximum outflow rate for some (a, c_r >= 0) -- see LpLamCand.
//   gain term  P_i = -(a + c_r E_{i+1}) E_{i+1}/dE_i = (-a) * alpha_i - c_r * beta_i     (needs a < 0)
//   loss term  Q_i =  (a + c_r E_i)     E_i/dE_i     =   a  * alpha'_i + c_r * beta'_i
// The maximiser of a linear function over a point set is a vertex of its convex hull; walking the
// hull over the admissible range of directions visits exactly the vertices that can win.
// Long-double arithmetic on the rounded table values.
// Gift wrapping, counter-clockwise from the rightmost (lowest) point, using orientation tests only.
// An edge (dx, dy) of the counter-clockwise hull has outward normal (dy, -dx): the direction at which
// its far end overtakes its near end.  The walk stops when that normal leaves the admissible cone:
// quarter = true: directions (u, v) with u >= 0, v >= 0;  quarter = false: v >= 0.
void hull_walk(const std::vector<long double> &px, const std::vector<long double> &py, bool quarter,
               std::vector<int> &out)
{
    const int n = (int)px.size();
    int cur = 0;
    for (int i = 1; i < n; ++i)
        if (px[i] > px[cur] || (px[i] == px[cur] && py[i] < py[cur])) cur = i;
    for (int guard = 0; guard <= n; ++guard) {
        out.push_back(cur);
        int nxt = -1;
        for (int j = 0; j < n; ++j) {
            if (j == cur || (px[j] == px[cur] && py[j] == py[cur])) continue;
            if (nxt < 0) { nxt = j; continue; }
            const long double ax = px[nxt] - px[cur], ay = py[nxt] - py[cur];
            const long double bx = px[j] - px[cur], by = py[j] - py[cur];
            const long double cr = ax * by - ay * bx;          // > 0: j is to the left of cur->nxt
            if (cr < 0.0L || (cr == 0.0L && bx * bx + by * by > ax * ax + ay * ay)) nxt = j;
        }
        if (nxt < 0) break;
        const long double dx = px[nxt] - px[cur], dy = py[nxt] - py[cur];
        if (dx > 0.0L || (quarter && dy < 0.0L)) break;        // normal (dy, -dx) left the cone
        cur = nxt;
    }
}

LpLamCand make_candidates(const std::vector<double> &E, const std::vector<double> &dE)
{
    const int nb = (int)dE.size();
    std::vector<long double> ax(nb), ay(nb), bx(nb), by(nb);
    for (int i = 0; i < nb; ++i) {
        const long double e0 = E[i], e1 = E[i + 1], d = dE[i];
        ax[i] = e1 / d;  ay[i] = -(e1 * e1 / d);      // gain: maximise (-a)*alpha - c_r*beta, (-a) > 0, c_r >= 0
        bx[i] = e0 / d;  by[i] = e0 * e0 / d;         // loss: maximise a*alpha' + c_r*beta', c_r >= 0, any a
    }
    std::vector<int> v;
    hull_walk(ax, ay, true, v);
    hull_walk(bx, by, false, v);
    v.push_back(0);
    v.push_back(nb - 1);
    std::sort(v.begin(), v.end());
    v.erase(std::unique(v.begin(), v.end()), v.end());
    LpLamCand c;
    std::memset(&c, 0, sizeof c);
    if ((int)v.size() > kLpMaxCand) { c.n = -1; return c; }
    c.n = (int)v.size();
    for (int k = 0; k < c.n; ++k) {
        c.bin[k] = v[k];
        c.el[k] = E[v[k]];
        c.er[k] = E[v[k] + 1];
        c.rde[k] = 1.0 / dE[v[k]];          // the same value as the device table's rdE
    }
    // On an exact log grid E_i/dE_i and E_{i+1}/dE_i do not depend on i, so the outflow rate is extremal
    // in an end bin; the table's rounding (E to 1 ulp, dE = E_{i+1} - E_i with cancellation) perturbs those
    // ratios by ~2^-53 E/dE.  64 times that, and never less than 1e-12.
    double worst = 0.0;
    for (int i = 0; i < nb; ++i) worst = std::max(worst, E[i + 1] / dE[i]);
    c.margin = std::max(1.0e-12, 64.0 * 1.1102230246251565e-16 * worst);
    return c;
}

bool nbins_ok(int nb) { return nb == 16 || nb == 32 || nb == 64 || nb == 128 || nb == 256 || nb == 512; }

int bit_length(unsigned long long v) { int b = 0; while (v) { ++b; v >>= 1; } return b; }

}  // namespace

struct lp_ctx {
    lp_config cfg;
    LpGeom geom;
    Layout lay;
    std::string err;
    int sm_count = 148;
    // bound buffers
    unsigned char *ws = nullptr;
    double *x = nullptr, *y = nullptr, *z = nullptr, *chi = nullptr;
    uint64_t *id = nullptr;
    int32_t *nsub_user = nullptr;
    double *lost_user = nullptr;
    double *eng = nullptr, *eng_scratch = nullptr;      // per-particle energy grid (lp_bind_energy_grid): moving-grid mode
    long long eng_capacity = 0;                         // rows the bound grid arrays hold
    bool eng_swapped = false;                           // (ping-pong) eng / eng_scratch have changed roles: the grid lives in
                                                        // the array bound as scratch
    // owned small tables
    double *tab = nullptr;                 // E[nb+1] | dE[nb] | rdE[nb]
    std::vector<double> h_edges, h_widths;
    LpLamCand cand;
    // state
    bool have_fields = false, stage0_done = false, spectra_done = false;
    int push_kind = 0;                     // which pusher ran stage 0: 1 two-stage (k1, x* kept), 2 three-stage (x0 kept)
    int rk3_next = 0;                      // next stage lp_push_rk3 expects
    bool status_valid = false;             // the status array describes the bound particles in their current order
    bool push_done = false;                // a pusher ran to its last stage since stage 0 (x^{n+1} is in place)
    bool cap_is_error = false;             // lp_set_cap_policy: lp_get_diag refuses a state with capped rows
    bool id_bits_stale = true;             // ids may have changed since id_bits was measured (bind, injection, host copy)
    int spectral_blocks[6] = { 0, 0, 0, 0, 0, 0 };   // resident blocks per SM of the spectral kernel variants [diag][mode], 0 = not set up
    long long capacity = 0;                // particles the workspace was sized for (cfg.np shrinks in lp_compact)
    int id_bits = 0, key_bits = 0;
    long long launches = 0, steps = 0, sorts = 0;
    // optional timing of the spectral kernel (lp_timing_enable): event pairs, resolved on read
    std::vector<cudaEvent_t> ev;
    size_t ev_used = 0;
    bool timing = false;
    // lp_step_host pipeline: copy-in and copy-out streams and their events (created on first use)
    cudaStream_t s_in = nullptr, s_out = nullptr;
    std::vector<cudaEvent_t> ev_pipe;

    // Two sets of particle arrays: 0 = the caller's bound arrays, 1 = their twins in the workspace (pos_alt,
    // alt_id, chi_alt; stride = capacity).  Without ping-pong (default) the state is always in set 0.  With it
    // (lp_set_pingpong) a re-sort reads one set through the permutation and writes the other, and `cur` flips.
    bool pingpong = false;
    int cur = 0;
    // particle exchange in progress (lp_migrate_count -> _pack -> _unpack): 0 none, 1 counted, 2 packed
    int mig_stage = 0;
    long long mig_left = 0, mig_right = 0;
    bool tile_configured = false;          // lp_interpolate_tile_kernel's shared-memory attribute is set
    bool split_records = false;            // cell records as two 32-byte arrays (dense sets) or one 64-byte array (LpCells)

    template <class T> T *at(size_t off) const { return reinterpret_cast<T *>(ws + off); }
    LpCells cells() const
    {
        const double4 *r = at<const double4>(lay.rec);
        if (split_records) return LpCells{ r, r + (size_t)cfg.nx * cfg.ny * cfg.nz, 1u };
        return LpCells{ r, r + 1, 2u };
    }
    struct Set { double *x, *y, *z; uint64_t *id; double *chi; };
    Set set(int which) const
    {
        if (which == 0) return Set{ x, y, z, id, chi };
        double *p = at<double>(lay.pos_alt);
        return Set{ p, p + capacity, p + 2 * capacity, at<uint64_t>(lay.alt_id), at<double>(lay.chi_alt) };
    }
    Set now() const { return set(cur); }
    Set other() const { return set(cur ^ 1); }
};

namespace {

lp_status fail(lp_ctx *c, lp_status st, const std::string &msg)
{
    if (c) c->err = msg;
    return st;
}

lp_status cuda_fail(lp_ctx *c, const char *what, cudaError_t e)
{
    return fail(c, LP_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define LP_CUDA(c, call)                                           \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail((c), #call, e_);   \
    } while (0)

lp_status count(lp_ctx *c, int n, const char *what)
{
    if (n < 0) {
        cudaError_t e = cudaGetLastError();
        return cuda_fail(c, what, e);
    }
    c->launches += n;
    return LP_OK;
}

lp_status validate(const lp_config *cfg, std::string &why)
{
    if (!cfg) { why = "cfg is NULL"; return LP_ERR_INVALID_ARG; }
    if (cfg->struct_size != sizeof(lp_config)) { why = "cfg->struct_size != sizeof(lp_config)"; return LP_ERR_INVALID_ARG; }
    if (cfg->nx < 1 || cfg->ny < 1 || cfg->nz < 1) { why = "grid size must be >= 1"; return LP_ERR_INVALID_ARG; }
    if ((long long)cfg->nx * cfg->ny * cfg->nz > (1ll << 31)) { why = "more than 2^31 cells"; return LP_ERR_UNSUPPORTED; }
    for (int d = 0; d < 3; ++d)
        if (!(cfg->xhi[d] > cfg->xlo[d])) { why = "xhi must exceed xlo"; return LP_ERR_INVALID_ARG; }
    if (cfg->np < 0 || cfg->np > 0xffffffffll) { why = "np out of range [0, 2^32)"; return LP_ERR_INVALID_ARG; }
    if (!nbins_ok(cfg->nbins)) { why = "nbins must be one of 16,32,64,128,256,512"; return LP_ERR_UNSUPPORTED; }
    if (!(cfg->e_min > 0.0) || !(cfg->e_max > cfg->e_min)) { why = "need 0 < e_min < e_max"; return LP_ERR_INVALID_ARG; }
    if (!(cfg->cfl_e > 0.0) || cfg->cfl_e > 1.0) { why = "need 0 < cfl_e <= 1"; return LP_ERR_INVALID_ARG; }
    if (cfg->max_substeps < 1) { why = "max_substeps must be >= 1"; return LP_ERR_INVALID_ARG; }
    if (cfg->sort_every < 0) { why = "sort_every must be >= 0"; return LP_ERR_INVALID_ARG; }
    if (!(cfg->kappa >= 0.0) || !(cfg->u_rad >= 0.0)) { why = "kappa and u_rad must be >= 0"; return LP_ERR_INVALID_ARG; }
    return LP_OK;
}

lp_status need_ready(lp_ctx *c, bool fields)
{
    if (!c) return LP_ERR_INVALID_ARG;
    if (!c->ws) return fail(c, LP_ERR_STATE, "no workspace bound (lp_bind_workspace)");
    if (c->cfg.np > 0 && !c->x) return fail(c, LP_ERR_STATE, "no particles bound (lp_bind_particles)");
    if (fields && !c->have_fields) return fail(c, LP_ERR_STATE, "fields not set (lp_set_fields)");
    return LP_OK;
}

// a bound energy grid must cover the capacity of the particle arrays (lp_rebind may have outgrown it)
lp_status grid_ok(lp_ctx *c)
{
    if (c->eng && c->eng_capacity < c->capacity)
        return fail(c, LP_ERR_STATE, "the energy-grid arrays hold fewer rows than the particle arrays (lp_rebind_energy_grid)");
    return LP_OK;
}

lp_status not_with_energy_grid(lp_ctx *c, const char *what)
{
    if (c->eng) return fail(c, LP_ERR_UNSUPPORTED, std::string(what) + " does not move the per-particle energy grid (lp_bind_energy_grid is active)");
    return LP_OK;
}

// spectral update on the per-particle moving grid (lp_moving.cu)
lp_status do_moving(lp_ctx *c, double dt, bool fused, cudaStream_t s, const uint32_t *perm = nullptr)
{
    lp_status gs = grid_ok(c);
    if (gs != LP_OK) return gs;
    const lp_ctx::Set n = c->now();
    LpMovingIO io{ n.x, n.y, n.z, c->eng, n.chi, n.x, n.y, n.z, c->eng, n.chi, nullptr, nullptr, nullptr };
    if (perm) {                         // re-sort folded into the step: read the current homes, write the other ones
        const lp_ctx::Set o = c->other();
        io = LpMovingIO{ n.x, n.y, n.z, c->eng, n.chi, o.x, o.y, o.z, c->eng_scratch, o.chi, perm, n.id, o.id };
    }
    const bool rec = c->timing && c->ev_used + 2 <= c->ev.size();
    if (rec) LP_CUDA(c, cudaEventRecord(c->ev[c->ev_used], s));
    lp_status st = count(c, lp_launch_moving(c->geom, c->cells(), io, c->at<double>(c->lay.rho_old),
                                             c->at<int32_t>(c->lay.status), fused, c->at<int32_t>(c->lay.nsub), c->nsub_user,
                                             c->cfg.np, c->cfg.nbins, dt, c->cfg.kappa, c->cfg.u_rad, c->sm_count, s),
                         "lp_moving_kernel launch");
    if (rec) {
        LP_CUDA(c, cudaEventRecord(c->ev[c->ev_used + 1], s));
        c->ev_used += 2;
    }
    if (st == LP_OK) {
        c->spectra_done = true;
        c->stage0_done = false; c->rk3_next = 0; c->push_done = false;
        if (fused) { c->status_valid = true; c->mig_stage = 0; }
        if (perm) {                     // the state now lives in the other homes
            c->cur ^= 1;
            std::swap(c->eng, c->eng_scratch);
            c->eng_swapped = !c->eng_swapped;
        }
    }
    return st;
}

LpPushArgs push_args(lp_ctx *c, double dt)
{
    LpPushArgs a;
    a.g = c->geom;
    a.cells = c->cells();
    const lp_ctx::Set n = c->now();
    a.x = n.x; a.y = n.y; a.z = n.z;
    a.k1 = c->at<double>(c->lay.k1);
    a.xs = c->at<double>(c->lay.xs);
    a.rho_old = c->at<double>(c->lay.rho_old);
    a.status = c->at<int32_t>(c->lay.status);
    a.np = c->cfg.np;
    a.dt = dt;
    return a;
}

// Where one launch of the spectral kernel reads and writes the particle arrays.
struct SpectralIO {
    const double *xin, *yin, *zin, *chi_in;
    double *x, *y, *z, *chi_out;
    const uint32_t *perm;              // re-sort folded into the fused step, or NULL
    const uint64_t *id_in;
    uint64_t *id_out;
};

SpectralIO io_in_place(const lp_ctx *c)
{
    const lp_ctx::Set n = c->now();
    return SpectralIO{ n.x, n.y, n.z, n.chi, n.x, n.y, n.z, n.chi, nullptr, nullptr, nullptr };
}

// p0, pcount: the particles [p0, p0 + pcount) only (pcount < 0: all)
lp_status do_spectral(lp_ctx *c, double dt, const SpectralIO &io, bool fused, cudaStream_t s,
                      long long p0 = 0, long long pcount = -1)
{
    LpSpectralArgs a;
    a.g = c->geom;
    a.cand = c->cand;
    a.status = c->at<int32_t>(c->lay.status);
    a.cells = c->cells();
    a.x = io.x; a.y = io.y; a.z = io.z;
    a.xin = io.xin; a.yin = io.yin; a.zin = io.zin;
    a.perm = io.perm; a.id_in = io.id_in; a.id_out = io.id_out;
    a.rho_old = c->at<double>(c->lay.rho_old);
    a.chi_in = io.chi_in;
    a.chi_out = io.chi_out;
    a.tab = c->tab;
    a.nsub_ws = c->at<int32_t>(c->lay.nsub);
    a.nsub_user = c->nsub_user;
    a.lost_ws = c->at<double>(c->lay.lost);
    a.lost_user = c->lost_user;
    a.np = c->cfg.np;
    if (pcount >= 0) {                  // a sub-range is the same launch on shifted arrays
        const size_t nb = (size_t)c->cfg.nbins;
        a.status += p0;
        a.x += p0; a.y += p0; a.z += p0;
        a.xin += p0; a.yin += p0; a.zin += p0;
        a.rho_old += p0;
        a.chi_in += (size_t)p0 * nb;
        a.chi_out += (size_t)p0 * nb;
        a.nsub_ws += p0;
        if (a.nsub_user) a.nsub_user += p0;
        a.lost_ws += p0;
        if (a.lost_user) a.lost_user += p0;
        a.np = pcount;
    }
    a.dt = dt;
    a.kappa = c->cfg.kappa;
    a.u_rad = c->cfg.u_rad;
    a.cfl_e = c->cfg.cfl_e;
    a.max_substeps = c->cfg.max_substeps;
    const bool rec = c->timing && c->ev_used + 2 <= c->ev.size();
    if (rec) LP_CUDA(c, cudaEventRecord(c->ev[c->ev_used], s));
    lp_status st = count(c, lp_launch_spectral(a, c->cfg.nbins, c->lost_user != nullptr, fused, c->sm_count,
                                                    c->spectral_blocks, s),
                         "lp_spectral_kernel launch");
    if (rec) {
        LP_CUDA(c, cudaEventRecord(c->ev[c->ev_used + 1], s));
        c->ev_used += 2;
    }
    if (st == LP_OK) {
        c->spectra_done = true;
        c->mig_stage = 0;                   // (the fused step moves the particles)
        c->stage0_done = false; c->rk3_next = 0; c->push_done = false;
        if (fused) c->status_valid = true;
    }
    return st;
}

// The permutation into (cell key, id) order of the current particles: perm[n] = index now of the n-th.
lp_status sort_permutation(lp_ctx *c, uint32_t **perm, cudaStream_t s)
{
    const long long np = c->cfg.np;
    const lp_ctx::Set n = c->now();
    LpSortBufs b;
    b.key = c->at<uint32_t>(c->lay.key);
    b.idx_a = c->at<uint32_t>(c->lay.idx_a);
    b.idx_b = c->at<uint32_t>(c->lay.idx_b);
    b.hist = c->at<uint32_t>(c->lay.hist);
    b.hist_elems = c->lay.hist_elems;
    b.digit = c->at<uint8_t>(c->lay.lost);          // the per-particle `lost` buffer is dead across a re-sort
    lp_status st;
    if (c->id_bits_stale) {
        // number of radix passes over the ids = bit length of the largest id among the current particles.
        // Measured on the caller's stream, once after every event that can change the ids (bind, raised
        // count, host copy); this is the one place a sort synchronises.
        unsigned long long *d = c->at<unsigned long long>(c->lay.maxid), h = 0;
        LP_CUDA(c, cudaMemsetAsync(d, 0, 8, s));
        if ((st = count(c, lp_launch_max_u64(n.id, np, d, s), "lp_max_u64_kernel launch")) != LP_OK) return st;
        LP_CUDA(c, cudaMemcpyAsync(&h, d, 8, cudaMemcpyDeviceToHost, s));
        LP_CUDA(c, cudaStreamSynchronize(s));
        c->id_bits = bit_length(h);
        c->id_bits_stale = false;
    }
    if (c->lay.counting) {
        // one counter per cell, rank counting inside the cells; the radix passes are enqueued behind it as a
        // fallback that runs only if a cell holds more than 64 particles (a flag on the device gates them)
        LpCountBufs cb;
        cb.cnt = c->at<uint32_t>(c->lay.cellcnt);
        cb.tile_sum = c->at<uint32_t>(c->lay.tile_sum);
        cb.seg_id = c->other().id;                 // scratch until the permuted ids are written there
        cb.overflow = c->at<uint32_t>(c->lay.maxid) + 2;
        return count(c, lp_launch_sort_perm_counting(c->geom, n.x, n.y, n.z, n.id, np, c->id_bits, c->key_bits, b, cb, perm, s),
                     "sort kernels launch");
    }
    return count(c, lp_launch_sort_perm(c->geom, n.x, n.y, n.z, n.id, np, c->id_bits, c->key_bits, b, perm, s),
                 "sort kernels launch");
}

void sort_invalidates(lp_ctx *c)
{
    c->stage0_done = false; c->rk3_next = 0; c->push_done = false;      // k1 / x* / rho_old refer to the old order
    c->spectra_done = false;     // so do the per-particle n_sub / lost of the last update
    c->status_valid = false;
    c->mig_stage = 0;
    ++c->sorts;
}

// Apply the permutation with the permute kernels.
//  * ping-pong: current set -> other set, which becomes the current one (no copy back).
//  * otherwise through scratch (x* buffer, alt_id, chi_alt).  in_place = true (lp_sort): everything is copied
//    back into the bound arrays.  in_place = false (lp_step without ping-pong): the ids go back, the permuted
//    positions stay in the x* scratch and the permuted rows in chi_alt for the fused kernel to read (it writes
//    the bound arrays), which saves four array copies; *io describes that launch.
lp_status do_sort(lp_ctx *c, bool in_place, SpectralIO *io, cudaStream_t s)
{
    const long long np = c->cfg.np;
    if (np == 0) return LP_OK;
    if (c->eng && !c->eng_scratch) return fail(c, LP_ERR_STATE, "a sort needs the eng_scratch array of lp_bind_energy_grid");
    if (grid_ok(c) != LP_OK) return LP_ERR_STATE;
    uint32_t *perm = nullptr;
    lp_status st = sort_permutation(c, &perm, s);
    if (st != LP_OK) return st;
    if (c->eng) {                       // the energy-grid rows follow their particles (through the scratch and back)
        const int len = c->cfg.nbins + 1;
        if ((st = count(c, lp_launch_permute_rows8(perm, c->eng, c->eng_scratch, np, len, s), "permute launch")) != LP_OK) return st;
        if (c->pingpong) {              // the scratch becomes the grid's home (lp_current_energy_grid)
            std::swap(c->eng, c->eng_scratch);
            c->eng_swapped = !c->eng_swapped;
        } else {
            LP_CUDA(c, cudaMemcpyAsync(c->eng, c->eng_scratch, (size_t)np * len * 8, cudaMemcpyDeviceToDevice, s));
        }
    }
    const lp_ctx::Set n = c->now();
    lp_ctx::Set o = c->other();
    if (!c->pingpong) {
        double *sx = c->at<double>(c->lay.xs);
        o = lp_ctx::Set{ sx, sx + np, sx + 2 * np, c->at<uint64_t>(c->lay.alt_id), c->at<double>(c->lay.chi_alt) };
    }
    const double *pos_src[3] = { n.x, n.y, n.z };
    double *pos_dst[3] = { o.x, o.y, o.z };
    for (int d = 0; d < 3; ++d)
        if ((st = count(c, lp_launch_permute_f64(perm, pos_src[d], pos_dst[d], np, s), "permute launch")) != LP_OK) return st;
    if ((st = count(c, lp_launch_permute_u64(perm, n.id, o.id, np, s), "permute launch")) != LP_OK) return st;
    if ((st = count(c, lp_launch_permute_rows(perm, n.chi, o.chi, np, c->cfg.nbins, s), "permute launch")) != LP_OK) return st;
    if (c->pingpong) {
        c->cur ^= 1;
    } else {
        LP_CUDA(c, cudaMemcpyAsync(n.id, o.id, (size_t)np * 8, cudaMemcpyDeviceToDevice, s));
        if (in_place) {
            for (int d = 0; d < 3; ++d)
                LP_CUDA(c, cudaMemcpyAsync(const_cast<double *>(pos_src[d]), pos_dst[d], (size_t)np * 8, cudaMemcpyDeviceToDevice, s));
            LP_CUDA(c, cudaMemcpyAsync(n.chi, o.chi, (size_t)np * c->cfg.nbins * 8, cudaMemcpyDeviceToDevice, s));
        } else if (io) {
            *io = SpectralIO{ o.x, o.y, o.z, o.chi, n.x, n.y, n.z, n.chi, nullptr, nullptr, nullptr };
        }
    }
    sort_invalidates(c);
    return LP_OK;
}

}  // namespace

extern "C" {

lp_status lp_create(const lp_config *cfg, lp_ctx **out)
{
    if (!out) return LP_ERR_INVALID_ARG;
    *out = nullptr;
    std::string why;
    lp_status st = validate(cfg, why);
    if (st != LP_OK) return st;
    lp_ctx *c = new (std::nothrow) lp_ctx();
    if (!c) return LP_ERR_INVALID_ARG;
    c->cfg = *cfg;
    c->capacity = cfg->np;
    c->lay = make_layout(*cfg);
#ifdef LP_FORCE_SPLIT_RECORDS               // (sweeps only)
    c->split_records = LP_FORCE_SPLIT_RECORDS != 0;
#else
    c->split_records = cfg->np >= (long long)cfg->nx * cfg->ny * cfg->nz;      // a particle or more per cell
#endif
    LpGeom &g = c->geom;
    g.nx = cfg->nx; g.ny = cfg->ny; g.nz = cfg->nz;
    const int n[3] = { cfg->nx, cfg->ny, cfg->nz };
    for (int d = 0; d < 3; ++d) {
        g.per[d] = cfg->periodic[d] ? 1 : 0;
        g.xlo[d] = cfg->xlo[d];
        g.xhi[d] = cfg->xhi[d];
        g.len[d] = cfg->xhi[d] - cfg->xlo[d];
        g.inv_dx[d] = (double)n[d] / (cfg->xhi[d] - cfg->xlo[d]);
    }
    c->key_bits = bit_length((unsigned long long)cfg->nx * cfg->ny * cfg->nz - 1ull);
    // bin table: N_b + 1 log-spaced edges on [e_min, e_max]
    const int nb = cfg->nbins;
    std::vector<double> tab((size_t)3 * nb + 1);
    for (int k = 0; k <= nb; ++k) tab[k] = cfg->e_min * std::pow(cfg->e_max / cfg->e_min, (double)k / (double)nb);
    for (int i = 0; i < nb; ++i) {
        tab[nb + 1 + i] = tab[i + 1] - tab[i];
        tab[2 * nb + 1 + i] = 1.0 / tab[nb + 1 + i];
    }
    c->h_edges.assign(tab.begin(), tab.begin() + nb + 1);
    c->h_widths.assign(tab.begin() + nb + 1, tab.begin() + 2 * nb + 1);
    c->cand = make_candidates(c->h_edges, c->h_widths);
    *out = c;
    LP_CUDA(c, cudaSetDevice(cfg->device));
    int sm = 0;
    LP_CUDA(c, cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, cfg->device));
    c->sm_count = sm > 0 ? sm : 148;
    LP_CUDA(c, cudaMalloc(&c->tab, tab.size() * sizeof(double)));
    LP_CUDA(c, cudaMemcpy(c->tab, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice));
    return LP_OK;
}

lp_status lp_destroy(lp_ctx *ctx)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    if (ctx->tab) cudaFree(ctx->tab);
    for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->ev_pipe) cudaEventDestroy(e);
    if (ctx->s_in) cudaStreamDestroy(ctx->s_in);
    if (ctx->s_out) cudaStreamDestroy(ctx->s_out);
    delete ctx;
    return LP_OK;
}

const char *lp_last_error(const lp_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

lp_status lp_workspace_bytes(const lp_config *cfg, size_t *out_bytes)
{
    if (!out_bytes) return LP_ERR_INVALID_ARG;
    std::string why;
    lp_status st = validate(cfg, why);
    if (st != LP_OK) return st;
    *out_bytes = make_layout(*cfg).total;
    return LP_OK;
}

lp_status lp_bind_workspace(lp_ctx *ctx, void *workspace, size_t bytes)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    if (!workspace) return fail(ctx, LP_ERR_WORKSPACE, "workspace is NULL");
    if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return fail(ctx, LP_ERR_WORKSPACE, "workspace not 256-byte aligned");
    if (bytes < ctx->lay.total) return fail(ctx, LP_ERR_WORKSPACE, "workspace smaller than lp_workspace_bytes");
    ctx->ws = static_cast<unsigned char *>(workspace);
    ctx->have_fields = false;
    ctx->stage0_done = false; ctx->rk3_next = 0; ctx->push_done = false;
    ctx->spectra_done = false;
    ctx->status_valid = false;
    return LP_OK;
}

lp_status lp_bind_particles(lp_ctx *ctx, double *x, double *y, double *z, uint64_t *id, double *chi)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    if (!ctx->ws) return fail(ctx, LP_ERR_STATE, "bind the workspace first");
    if (ctx->cfg.np > 0 && (!x || !y || !z || !id || !chi)) return fail(ctx, LP_ERR_INVALID_ARG, "NULL particle array");
    if (reinterpret_cast<uintptr_t>(chi) % 16) return fail(ctx, LP_ERR_INVALID_ARG, "chi not 16-byte aligned");
    ctx->x = x; ctx->y = y; ctx->z = z; ctx->id = id; ctx->chi = chi;
    ctx->cur = 0;                       // the state is what the caller just bound
    ctx->mig_stage = 0;
    ctx->stage0_done = false; ctx->rk3_next = 0; ctx->push_done = false;
    ctx->spectra_done = false;
    ctx->status_valid = false;
    ctx->id_bits = 0;
    ctx->id_bits_stale = true;          // measured on the caller's stream by the next sort
    return LP_OK;
}

lp_status lp_bind_diag(lp_ctx *ctx, int32_t *nsub, double *lost)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    ctx->nsub_user = nsub;
    ctx->lost_user = lost;
    return LP_OK;
}

lp_status lp_set_fields(lp_ctx *ctx, const double *vx, const double *vy, const double *vz, const double *bx,
                        const double *by, const double *bz, const double *rho, void *stream)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    if (!ctx->ws) return fail(ctx, LP_ERR_STATE, "no workspace bound (lp_bind_workspace)");
    if (!vx || !vy || !vz || !bx || !by || !bz || !rho) return fail(ctx, LP_ERR_INVALID_ARG, "NULL field array");
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    const double *f[7] = { vx, vy, vz, bx, by, bz, rho };
    const long long ncell = (long long)ctx->cfg.nx * ctx->cfg.ny * ctx->cfg.nz;
    const LpCells cl = ctx->cells();
    lp_status st = count(ctx, lp_launch_repack(f, const_cast<double4 *>(cl.recA), const_cast<double4 *>(cl.recB), cl.stride, ncell,
                                               static_cast<cudaStream_t>(stream)), "lp_repack_kernel launch");
    if (st == LP_OK) ctx->have_fields = true;
    return st;
}

lp_status lp_interpolate(lp_ctx *ctx, double *out7, uint32_t *cell_key, void *stream)
{
    lp_status st = need_ready(ctx, out7 != nullptr);
    if (st != LP_OK) return st;
    if (!out7 && !cell_key) return LP_OK;
    if (ctx->cfg.np == 0) return LP_OK;
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    const lp_ctx::Set n = ctx->now();
    return count(ctx, lp_launch_interpolate(ctx->geom, ctx->cells(), n.x, n.y, n.z, ctx->cfg.np, out7, cell_key,
                                            static_cast<cudaStream_t>(stream)), "lp_interpolate_kernel launch");
}

lp_status lp_interpolate_tiled(lp_ctx *ctx, double *out7, void *stream)
{
    lp_status st = need_ready(ctx, true);
    if (st != LP_OK) return st;
    if (!out7) return fail(ctx, LP_ERR_INVALID_ARG, "out7 is NULL");
    if (ctx->cfg.np == 0) return LP_OK;
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    const lp_ctx::Set n = ctx->now();
    return count(ctx, lp_launch_interpolate_tiled(ctx->geom, ctx->cells(), n.x, n.y, n.z, ctx->cfg.np, out7,
                                                  &ctx->tile_configured, static_cast<cudaStream_t>(stream)), "lp_interpolate_tile_kernel launch");
}

lp_status lp_sort(lp_ctx *ctx, void *stream)
{
    lp_status st = need_ready(ctx, false);
    if (st != LP_OK) return st;
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    return do_sort(ctx, true, nullptr, static_cast<cudaStream_t>(stream));
}

lp_status lp_push(lp_ctx *ctx, double dt, int stage, void *stream)
{
    lp_status st = need_ready(ctx, true);
    if (st != LP_OK) return st;
    if (stage != 0 && stage != 1) return fail(ctx, LP_ERR_INVALID_ARG, "stage must be 0 or 1");
    if (stage == 1 && !(ctx->stage0_done && ctx->push_kind == 1)) return fail(ctx, LP_ERR_STATE, "lp_push stage 1 without stage 0");
    if (ctx->cfg.np == 0) { ctx->stage0_done = true; ctx->push_kind = 1; ctx->push_done = stage == 1; return LP_OK; }
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    LpPushArgs a = push_args(ctx, dt);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (stage == 0) {
        st = count(ctx, lp_launch_push0(a, s), "lp_push0_kernel launch");
        if (st == LP_OK) { ctx->stage0_done = true; ctx->push_kind = 1; ctx->rk3_next = 0; ctx->push_done = false; }
        return st;
    }
    st = count(ctx, lp_launch_push1(a, s), "lp_push1_kernel launch");
    if (st == LP_OK) { ctx->status_valid = true; ctx->push_done = true; ctx->mig_stage = 0; }
    return st;
}

lp_status lp_push_rk3(lp_ctx *ctx, double dt, int stage, void *stream)
{
    lp_status st = need_ready(ctx, true);
    if (st != LP_OK) return st;
    if (stage < 0 || stage > 2) return fail(ctx, LP_ERR_INVALID_ARG, "stage must be 0, 1 or 2");
    if (stage != 0 && !(ctx->push_kind == 2 && ctx->rk3_next == stage))
        return fail(ctx, LP_ERR_STATE, "lp_push_rk3 stages must run in the order 0, 1, 2");
    if (ctx->cfg.np > 0) {
        LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
        LpPushArgs a = push_args(ctx, dt);
        st = count(ctx, lp_launch_push_rk3(a, stage, static_cast<cudaStream_t>(stream)), "lp_push_rk3_kernel launch");
        if (st != LP_OK) return st;
    }
    ctx->mig_stage = 0;                 // every stage writes the bound positions
    if (stage == 0) { ctx->stage0_done = true; ctx->push_kind = 2; ctx->status_valid = false; ctx->push_done = false; }
    if (stage == 2) { ctx->status_valid = true; ctx->push_done = true; }
    ctx->rk3_next = stage == 2 ? 0 : stage + 1;
    return LP_OK;
}

lp_status lp_spectral_update(lp_ctx *ctx, double dt, void *stream)
{
    lp_status st = need_ready(ctx, true);
    if (st != LP_OK) return st;
    if (!ctx->stage0_done) return fail(ctx, LP_ERR_STATE, "lp_spectral_update needs rho_old of lp_push stage 0");
    if (!ctx->push_done)
        return fail(ctx, LP_ERR_STATE, "lp_spectral_update needs the push finished (lp_push stage 1 / lp_push_rk3 stage 2)");
    if (ctx->cfg.np == 0) return LP_OK;
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    if (ctx->eng) return do_moving(ctx, dt, false, static_cast<cudaStream_t>(stream));
    return do_spectral(ctx, dt, io_in_place(ctx), false, static_cast<cudaStream_t>(stream));
}

lp_status lp_shock_update(lp_ctx *ctx, const double *r, double q_r, void *stream)
{
    lp_status st = need_ready(ctx, false);
    if (st != LP_OK) return st;
    if ((st = grid_ok(ctx)) != LP_OK) return st;
    if (ctx->cfg.np == 0) return LP_OK;
    if (!r) return fail(ctx, LP_ERR_INVALID_ARG, "r is NULL");
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    return count(ctx, lp_launch_shock(ctx->tab, ctx->eng, r, q_r, ctx->now().chi, ctx->cfg.np, ctx->cfg.nbins, ctx->sm_count,
                                      static_cast<cudaStream_t>(stream)), "lp_shock_kernel launch");
}

lp_status lp_compact(lp_ctx *ctx, const int32_t *flag, int64_t *np_new, void *stream)
{
    lp_status st = need_ready(ctx, false);
    if (st != LP_OK) return st;
    if (!np_new) return fail(ctx, LP_ERR_INVALID_ARG, "np_new is NULL");
    *np_new = ctx->cfg.np;
    if (ctx->cfg.np == 0) return LP_OK;
    if ((st = grid_ok(ctx)) != LP_OK) return st;
    if (!flag && !ctx->status_valid)
        return fail(ctx, LP_ERR_STATE, "no flags given and no outside-box status of the bound particles (lp_push 1 / lp_step first)");
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (!flag) flag = ctx->at<int32_t>(ctx->lay.status);
    unsigned long long *counts = ctx->at<unsigned long long>(ctx->lay.partial), h_counts[2] = { 0, 0 };
    st = count(ctx, lp_launch_compact(flag, ctx->cfg.np, ctx->cfg.nbins, ctx->at<uint32_t>(ctx->lay.hist),
                                      ctx->at<uint32_t>(ctx->lay.idx_a), ctx->at<uint32_t>(ctx->lay.idx_b),
                                      ctx->at<uint32_t>(ctx->lay.key), counts, ctx->now().x, ctx->now().y, ctx->now().z,
                                      ctx->now().id, ctx->now().chi, ctx->eng, ctx->sm_count, s), "compaction kernels launch");
    if (st != LP_OK) return st;
    LP_CUDA(ctx, cudaMemcpyAsync(h_counts, counts, sizeof h_counts, cudaMemcpyDeviceToHost, s));
    LP_CUDA(ctx, cudaStreamSynchronize(s));
    ctx->cfg.np -= (long long)h_counts[0];          // the workspace keeps its size (capacity)
    ctx->mig_stage = 0;
    ctx->stage0_done = false; ctx->rk3_next = 0; ctx->push_done = false;
    ctx->spectra_done = false;
    ctx->status_valid = false;
    *np_new = ctx->cfg.np;
    return LP_OK;
}

lp_status lp_chunked_capacity(int64_t n, int32_t e, int64_t *capacity)
{
    if (!capacity || n < 0 || e < 0 || e > 40) return LP_ERR_INVALID_ARG;
    const int64_t len = (int64_t)1 << e;
    const int64_t nc = (n >> e) + (n % len == 0 ? 0 : 1);          // Listing 1
    *capacity = nc << e;
    return LP_OK;
}

lp_status lp_set_count(lp_ctx *ctx, int64_t np_new)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    if (np_new < 0 || np_new > ctx->capacity) return fail(ctx, LP_ERR_INVALID_ARG, "count outside [0, capacity of lp_create]");
    if (np_new > 0 && ctx->ws && !ctx->x) return fail(ctx, LP_ERR_STATE, "no particles bound (lp_bind_particles)");
    if (np_new > ctx->cfg.np) ctx->id_bits_stale = true;      // injected particles bring their own ids
    ctx->cfg.np = np_new;
    ctx->mig_stage = 0;
    ctx->stage0_done = false; ctx->rk3_next = 0; ctx->push_done = false;
    ctx->spectra_done = false;
    ctx->status_valid = false;
    return LP_OK;
}

lp_status lp_capacity(const lp_ctx *ctx, int64_t *capacity)
{
    if (!ctx || !capacity) return LP_ERR_INVALID_ARG;
    *capacity = ctx->capacity;
    return LP_OK;
}

lp_status lp_workspace_bytes_for(const lp_ctx *ctx, int64_t capacity, size_t *out_bytes)
{
    if (!ctx || !out_bytes || capacity < 0 || capacity > 0xffffffffll) return LP_ERR_INVALID_ARG;
    lp_config c = ctx->cfg;
    c.np = capacity;
    *out_bytes = make_layout(c).total;
    return LP_OK;
}

lp_status lp_rebind(lp_ctx *ctx, int64_t capacity, void *workspace, size_t bytes, double *x, double *y, double *z,
                    uint64_t *id, double *chi, void *stream)
{
    lp_status st = need_ready(ctx, false);
    if (st != LP_OK) return st;
    if (capacity < ctx->cfg.np || capacity > 0xffffffffll) return fail(ctx, LP_ERR_INVALID_ARG, "capacity below the particle count or >= 2^32");
    if (capacity > 0 && (!x || !y || !z || !id || !chi)) return fail(ctx, LP_ERR_INVALID_ARG, "NULL particle array");
    if (reinterpret_cast<uintptr_t>(chi) % 16) return fail(ctx, LP_ERR_INVALID_ARG, "chi not 16-byte aligned");
    if (!workspace) return fail(ctx, LP_ERR_WORKSPACE, "workspace is NULL");
    if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return fail(ctx, LP_ERR_WORKSPACE, "workspace not 256-byte aligned");
    lp_config ncfg = ctx->cfg;
    ncfg.np = capacity;
    const Layout nl = make_layout(ncfg);
    if (bytes < nl.total) return fail(ctx, LP_ERR_WORKSPACE, "workspace smaller than lp_workspace_bytes_for(capacity)");
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    unsigned char *nws = static_cast<unsigned char *>(workspace);
    const size_t np = (size_t)ctx->cfg.np, nb = (size_t)ctx->cfg.nbins;
    const lp_ctx::Set n = ctx->now();
    if (np) {
        LP_CUDA(ctx, cudaMemcpyAsync(x, n.x, np * 8, cudaMemcpyDeviceToDevice, s));
        LP_CUDA(ctx, cudaMemcpyAsync(y, n.y, np * 8, cudaMemcpyDeviceToDevice, s));
        LP_CUDA(ctx, cudaMemcpyAsync(z, n.z, np * 8, cudaMemcpyDeviceToDevice, s));
        LP_CUDA(ctx, cudaMemcpyAsync(id, n.id, np * 8, cudaMemcpyDeviceToDevice, s));
        LP_CUDA(ctx, cudaMemcpyAsync(chi, n.chi, np * nb * 8, cudaMemcpyDeviceToDevice, s));
    }
    if (ctx->have_fields)
        LP_CUDA(ctx, cudaMemcpyAsync(nws + nl.rec, ctx->ws + ctx->lay.rec, (size_t)ctx->cfg.nx * ctx->cfg.ny * ctx->cfg.nz * 64,
                                     cudaMemcpyDeviceToDevice, s));
    if (ctx->mig_stage == 2) {          // an exchange is under way: its hole list moves along
        const size_t nholes = (size_t)(ctx->mig_left + ctx->mig_right);
        if (nholes) LP_CUDA(ctx, cudaMemcpyAsync(nws + nl.idx_a, ctx->ws + ctx->lay.idx_a, nholes * 4, cudaMemcpyDeviceToDevice, s));
    } else {
        ctx->mig_stage = 0;
    }
    ctx->ws = nws;
    ctx->lay = nl;
    ctx->capacity = capacity;
    ctx->x = x; ctx->y = y; ctx->z = z; ctx->id = id; ctx->chi = chi;
    ctx->cur = 0;
    ctx->nsub_user = nullptr;
    ctx->lost_user = nullptr;
    ctx->stage0_done = false; ctx->rk3_next = 0; ctx->push_done = false;
    ctx->spectra_done = false;
    ctx->status_valid = false;
    return LP_OK;
}

lp_status lp_set_pingpong(lp_ctx *ctx, int enable, void *stream)
{
    lp_status st = need_ready(ctx, false);
    if (st != LP_OK) return st;
    if (!enable && ctx->cur != 0 && ctx->cfg.np > 0) {        // bring the state home to the bound arrays
        LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
        cudaStream_t s = static_cast<cudaStream_t>(stream);
        const lp_ctx::Set n = ctx->now(), b = ctx->set(0);
        const size_t np = (size_t)ctx->cfg.np;
        LP_CUDA(ctx, cudaMemcpyAsync(b.x, n.x, np * 8, cudaMemcpyDeviceToDevice, s));
        LP_CUDA(ctx, cudaMemcpyAsync(b.y, n.y, np * 8, cudaMemcpyDeviceToDevice, s));
        LP_CUDA(ctx, cudaMemcpyAsync(b.z, n.z, np * 8, cudaMemcpyDeviceToDevice, s));
        LP_CUDA(ctx, cudaMemcpyAsync(b.id, n.id, np * 8, cudaMemcpyDeviceToDevice, s));
        LP_CUDA(ctx, cudaMemcpyAsync(b.chi, n.chi, np * (size_t)ctx->cfg.nbins * 8, cudaMemcpyDeviceToDevice, s));
    }
    if (!enable && ctx->eng && ctx->eng_swapped) {           // the grid goes home to the array bound as eng
        LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
        if (ctx->cfg.np > 0)
            LP_CUDA(ctx, cudaMemcpyAsync(ctx->eng_scratch, ctx->eng, (size_t)ctx->cfg.np * (ctx->cfg.nbins + 1) * 8,
                                         cudaMemcpyDeviceToDevice, static_cast<cudaStream_t>(stream)));
        std::swap(ctx->eng, ctx->eng_scratch);
        ctx->eng_swapped = false;
    }
    if (!enable) ctx->cur = 0;
    ctx->pingpong = enable != 0;
    return LP_OK;
}

lp_status lp_current_particles(const lp_ctx *ctx, double **x, double **y, double **z, uint64_t **id, double **chi)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    if (!ctx->ws || (ctx->cfg.np > 0 && !ctx->x)) return LP_ERR_STATE;
    const lp_ctx::Set n = ctx->now();
    if (x) *x = n.x;
    if (y) *y = n.y;
    if (z) *z = n.z;
    if (id) *id = n.id;
    if (chi) *chi = n.chi;
    return LP_OK;
}

lp_status lp_migrate_record_bytes(const lp_ctx *ctx, size_t *bytes)
{
    if (!ctx || !bytes) return LP_ERR_INVALID_ARG;
    *bytes = 32 + 8 * (size_t)ctx->cfg.nbins + (ctx->eng ? 8 * ((size_t)ctx->cfg.nbins + 1) : 0);
    return LP_OK;
}

lp_status lp_migrate_count(lp_ctx *ctx, int axis, double lo, double hi, int64_t *n_left, int64_t *n_right, void *stream)
{
    lp_status st = need_ready(ctx, false);
    if (st != LP_OK) return st;
    if (axis < 0 || axis > 2 || !n_left || !n_right || !(hi > lo)) return fail(ctx, LP_ERR_INVALID_ARG, "bad axis, interval or NULL output");
    if ((st = grid_ok(ctx)) != LP_OK) return st;
    ctx->mig_stage = 0;
    *n_left = *n_right = 0;
    ctx->mig_left = ctx->mig_right = 0;
    if (ctx->cfg.np > 0) {
        LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
        cudaStream_t s = static_cast<cudaStream_t>(stream);
        const lp_ctx::Set n = ctx->now();
        const double *pos = axis == 0 ? n.x : (axis == 1 ? n.y : n.z);
        unsigned long long *counts = ctx->at<unsigned long long>(ctx->lay.partial), h[2] = { 0, 0 };
        st = count(ctx, lp_launch_migrate_count(pos, ctx->cfg.np, lo, hi, ctx->geom.len[axis], ctx->geom.per[axis],
                                                ctx->at<uint32_t>(ctx->lay.key), ctx->at<unsigned long long>(ctx->lay.hist), counts,
                                                ctx->at<uint32_t>(ctx->lay.idx_a), ctx->at<uint32_t>(ctx->lay.idx_b), s),
                   "exchange count kernels launch");
        if (st != LP_OK) return st;
        LP_CUDA(ctx, cudaMemcpyAsync(h, counts, sizeof h, cudaMemcpyDeviceToHost, s));
        LP_CUDA(ctx, cudaStreamSynchronize(s));
        ctx->mig_left = (long long)h[0];
        ctx->mig_right = (long long)h[1];
    }
    *n_left = ctx->mig_left;
    *n_right = ctx->mig_right;
    ctx->mig_stage = 1;
    return LP_OK;
}

lp_status lp_migrate_pack(lp_ctx *ctx, void *buf_left, void *buf_right, void *stream)
{
    lp_status st = need_ready(ctx, false);
    if (st != LP_OK) return st;
    if (ctx->mig_stage != 1) return fail(ctx, LP_ERR_STATE, "lp_migrate_pack needs lp_migrate_count first");
    if ((ctx->mig_left > 0 && !buf_left) || (ctx->mig_right > 0 && !buf_right)) return fail(ctx, LP_ERR_INVALID_ARG, "NULL send buffer");
    if (reinterpret_cast<uintptr_t>(buf_left) % 16 || reinterpret_cast<uintptr_t>(buf_right) % 16)
        return fail(ctx, LP_ERR_INVALID_ARG, "send buffer not 16-byte aligned");
    const long long nleave = ctx->mig_left + ctx->mig_right;
    if (nleave > 0) {
        LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
        const lp_ctx::Set n = ctx->now();
        st = count(ctx, lp_launch_migrate_pack(ctx->mig_left, ctx->mig_right, ctx->at<uint32_t>(ctx->lay.idx_b),
                                               n.x, n.y, n.z, n.id, n.chi, ctx->eng, ctx->cfg.nbins, buf_left, buf_right, ctx->sm_count,
                                               static_cast<cudaStream_t>(stream)), "exchange pack kernel launch");
        if (st != LP_OK) return st;
    }
    ctx->mig_stage = 2;
    return LP_OK;
}

lp_status lp_migrate_unpack(lp_ctx *ctx, const void *from_left, int64_t n_from_left, const void *from_right,
                            int64_t n_from_right, int64_t *np_new, void *stream)
{
    lp_status st = need_ready(ctx, false);
    if (st != LP_OK) return st;
    if (!np_new) return fail(ctx, LP_ERR_INVALID_ARG, "np_new is NULL");
    *np_new = ctx->cfg.np;
    if (ctx->mig_stage != 2) return fail(ctx, LP_ERR_STATE, "lp_migrate_unpack needs lp_migrate_pack first");
    if (n_from_left < 0 || n_from_right < 0 || (n_from_left > 0 && !from_left) || (n_from_right > 0 && !from_right))
        return fail(ctx, LP_ERR_INVALID_ARG, "bad receive buffer");
    if (reinterpret_cast<uintptr_t>(from_left) % 16 || reinterpret_cast<uintptr_t>(from_right) % 16)
        return fail(ctx, LP_ERR_INVALID_ARG, "receive buffer not 16-byte aligned");
    const long long np = ctx->cfg.np, nholes = ctx->mig_left + ctx->mig_right, nin = n_from_left + n_from_right;
    const long long grown = np + (nin > nholes ? nin - nholes : 0);
    if (grown > ctx->capacity)
        return fail(ctx, LP_ERR_WORKSPACE, "arrivals exceed the capacity of the particle arrays (lp_rebind to grow)");
    if ((st = grid_ok(ctx)) != LP_OK) return st;
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const lp_ctx::Set n = ctx->now();
    int32_t *flag = ctx->at<int32_t>(ctx->lay.nsub);          // (per-particle n_sub is invalidated below anyway)
    const bool rest = nin < nholes;
    if (rest) LP_CUDA(ctx, cudaMemsetAsync(flag, 0, (size_t)np * 4, s));
    if (nin > 0 || rest) {
        st = count(ctx, lp_launch_migrate_unpack(from_left, n_from_left, from_right, n_from_right, ctx->at<uint32_t>(ctx->lay.idx_a),
                                                 nholes, np, n.x, n.y, n.z, n.id, n.chi, ctx->eng, ctx->cfg.nbins, rest ? flag : nullptr,
                                                 ctx->sm_count, s), "exchange unpack kernels launch");
        if (st != LP_OK) return st;
    }
    ctx->mig_stage = 0;
    ctx->cfg.np = grown;
    ctx->id_bits_stale = true;                                // arrivals bring their own ids
    ctx->stage0_done = false; ctx->rk3_next = 0; ctx->push_done = false;
    ctx->spectra_done = false;
    ctx->status_valid = false;
    if (rest) {                                               // holes no arrival filled: the compaction of Section 3.2
        int64_t after = 0;
        if ((st = lp_compact(ctx, flag, &after, stream)) != LP_OK) return st;
    }
    *np_new = ctx->cfg.np;
    return LP_OK;
}

lp_status lp_bind_energy_grid(lp_ctx *ctx, double *eng, double *eng_scratch)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    if (!eng && eng_scratch) return fail(ctx, LP_ERR_INVALID_ARG, "eng_scratch without eng");
    if (eng && ctx->cur != 0) return fail(ctx, LP_ERR_STATE, "bind the energy grid while the state is in the bound arrays");
    ctx->eng = eng;
    ctx->eng_scratch = eng_scratch;
    ctx->eng_swapped = false;
    ctx->eng_capacity = eng ? ctx->capacity : 0;
    ctx->spectra_done = false;
    return LP_OK;
}

lp_status lp_current_energy_grid(const lp_ctx *ctx, double **eng)
{
    if (!ctx || !eng) return LP_ERR_INVALID_ARG;
    *eng = ctx->eng;
    return LP_OK;
}

lp_status lp_rebind_energy_grid(lp_ctx *ctx, double *eng, double *eng_scratch, void *stream)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    if (!ctx->eng) return fail(ctx, LP_ERR_STATE, "no energy grid bound (lp_bind_energy_grid)");
    if (!eng) return fail(ctx, LP_ERR_INVALID_ARG, "eng is NULL");
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    if (ctx->cfg.np > 0 && eng != ctx->eng)
        LP_CUDA(ctx, cudaMemcpyAsync(eng, ctx->eng, (size_t)ctx->cfg.np * (ctx->cfg.nbins + 1) * 8, cudaMemcpyDeviceToDevice,
                                     static_cast<cudaStream_t>(stream)));
    ctx->eng = eng;
    ctx->eng_scratch = eng_scratch;
    ctx->eng_swapped = false;
    ctx->eng_capacity = ctx->capacity;
    return LP_OK;
}

lp_status lp_init_energy_grid(lp_ctx *ctx, int64_t first, int64_t count_, void *stream)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    if (!ctx->eng) return fail(ctx, LP_ERR_STATE, "no energy grid bound (lp_bind_energy_grid)");
    if (first < 0 || count_ < 0 || first + count_ > ctx->eng_capacity) return fail(ctx, LP_ERR_INVALID_ARG, "rows outside the grid arrays");
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    return count(ctx, lp_launch_moving_init(ctx->tab, ctx->cfg.nbins, ctx->eng, first, count_, static_cast<cudaStream_t>(stream)),
                 "lp_moving_init_kernel launch");
}

lp_status lp_step(lp_ctx *ctx, double dt, void *stream)
{
    lp_status st = need_ready(ctx, true);
    if (st != LP_OK) return st;
    ++ctx->steps;
    if (ctx->cfg.np == 0) return LP_OK;
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const bool sort_now = ctx->cfg.sort_every > 0 && (ctx->steps - 1) % ctx->cfg.sort_every == 0;
    if (ctx->eng) {
        // moving energy grid: one kernel that does both push stages and the grid update; on a re-sort step with
        // ping-pong buffers it also reads everything through the permutation (else the rows are permuted first)
        if (sort_now && ctx->pingpong && ctx->eng_scratch) {
            if ((st = grid_ok(ctx)) != LP_OK) return st;
            uint32_t *perm = nullptr;
            if ((st = sort_permutation(ctx, &perm, s)) != LP_OK) return st;
            sort_invalidates(ctx);
            return do_moving(ctx, dt, true, s, perm);
        }
        if (sort_now && (st = do_sort(ctx, true, nullptr, s)) != LP_OK) return st;
        return do_moving(ctx, dt, true, s);
    }
    SpectralIO io = io_in_place(ctx);
    bool flip = false;
    if (sort_now && ctx->pingpong) {
        // the re-sort is folded into the fused kernel: it reads the current set through the permutation
        // and writes the other set in the new order -- no permute pass, no copy back
        uint32_t *perm = nullptr;
        if ((st = sort_permutation(ctx, &perm, s)) != LP_OK) return st;
        const lp_ctx::Set n = ctx->now(), o = ctx->other();
        io = SpectralIO{ n.x, n.y, n.z, n.chi, o.x, o.y, o.z, o.chi, perm, n.id, o.id };
        sort_invalidates(ctx);
        flip = true;
    } else if (sort_now) {
        // the permuted rows and positions stay in the workspace; the fused kernel reads them from there
        // and writes the bound arrays
        if ((st = do_sort(ctx, false, &io, s)) != LP_OK) return st;
    }
    // frozen fields: both push stages run inside the spectral kernel's per-particle phase
    st = do_spectral(ctx, dt, io, true, s);
    if (st == LP_OK && flip) ctx->cur ^= 1;
    return st;
}

lp_status lp_step_host(lp_ctx *ctx, double dt, double *hx, double *hy, double *hz, uint64_t *hid, double *hchi,
                       void *stream)
{
    lp_status st = need_ready(ctx, true);
    if (st != LP_OK) return st;
    if ((st = not_with_energy_grid(ctx, "lp_step_host")) != LP_OK) return st;
    if (ctx->cfg.np > 0 && (!hx || !hy || !hz || !hid || !hchi)) return fail(ctx, LP_ERR_INVALID_ARG, "NULL host array");
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const size_t np = (size_t)ctx->cfg.np, nb = (size_t)ctx->cfg.nbins;
    const bool sort_now = ctx->cfg.sort_every > 0 && ctx->steps % ctx->cfg.sort_every == 0;
    constexpr int kBatches = 16;
    constexpr size_t kMinPipelined = (size_t)1 << 16;        // below this the copies are latency, not bandwidth
    if (np < kMinPipelined || sort_now) {
        // whole arrays in, one lp_step, whole arrays out (a re-sort needs every row on the device first)
        if (np) {
            const lp_ctx::Set n = ctx->now();
            LP_CUDA(ctx, cudaMemcpyAsync(n.x, hx, np * 8, cudaMemcpyHostToDevice, s));
            LP_CUDA(ctx, cudaMemcpyAsync(n.y, hy, np * 8, cudaMemcpyHostToDevice, s));
            LP_CUDA(ctx, cudaMemcpyAsync(n.z, hz, np * 8, cudaMemcpyHostToDevice, s));
            LP_CUDA(ctx, cudaMemcpyAsync(n.id, hid, np * 8, cudaMemcpyHostToDevice, s));
            LP_CUDA(ctx, cudaMemcpyAsync(n.chi, hchi, np * nb * 8, cudaMemcpyHostToDevice, s));
            ctx->id_bits_stale = true;                  // the host may hand in other ids than last time
        }
        if ((st = lp_step(ctx, dt, stream)) != LP_OK) return st;
        if (np) {
            const lp_ctx::Set n = ctx->now();            // (a folded re-sort has moved the state to the other set)
            LP_CUDA(ctx, cudaMemcpyAsync(hx, n.x, np * 8, cudaMemcpyDeviceToHost, s));
            LP_CUDA(ctx, cudaMemcpyAsync(hy, n.y, np * 8, cudaMemcpyDeviceToHost, s));
            LP_CUDA(ctx, cudaMemcpyAsync(hz, n.z, np * 8, cudaMemcpyDeviceToHost, s));
            LP_CUDA(ctx, cudaMemcpyAsync(hid, n.id, np * 8, cudaMemcpyDeviceToHost, s));
            LP_CUDA(ctx, cudaMemcpyAsync(hchi, n.chi, np * nb * 8, cudaMemcpyDeviceToHost, s));
        }
        LP_CUDA(ctx, cudaStreamSynchronize(s));
        return LP_OK;
    }

    // Pipelined: particles are independent, so the step runs batch by batch while the rows of the next
    // batch come in (copy-in stream) and those of the previous one go out (copy-out stream): the two
    // PCIe directions and the kernels overlap.  Batch boundaries are multiples of 32 particles.
    if (!ctx->s_in) {
        LP_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->s_in, cudaStreamNonBlocking));
        LP_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->s_out, cudaStreamNonBlocking));
        for (int i = 0; i < 2 * kBatches + 2; ++i) {
            cudaEvent_t e;
            LP_CUDA(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            ctx->ev_pipe.push_back(e);
        }
    }
    const lp_ctx::Set n = ctx->now();
    cudaEvent_t *ev_in = ctx->ev_pipe.data(), *ev_k = ev_in + kBatches;
    cudaEvent_t ev_start = ctx->ev_pipe[2 * kBatches], ev_done = ctx->ev_pipe[2 * kBatches + 1];
    const size_t per = ((np + kBatches - 1) / kBatches + 31) / 32 * 32;
    LP_CUDA(ctx, cudaEventRecord(ev_start, s));                 // copies start after earlier work on s
    LP_CUDA(ctx, cudaStreamWaitEvent(ctx->s_in, ev_start, 0));
    LP_CUDA(ctx, cudaStreamWaitEvent(ctx->s_out, ev_start, 0));
    LP_CUDA(ctx, cudaMemcpyAsync(n.x, hx, np * 8, cudaMemcpyHostToDevice, ctx->s_in));
    LP_CUDA(ctx, cudaMemcpyAsync(n.y, hy, np * 8, cudaMemcpyHostToDevice, ctx->s_in));
    LP_CUDA(ctx, cudaMemcpyAsync(n.z, hz, np * 8, cudaMemcpyHostToDevice, ctx->s_in));
    LP_CUDA(ctx, cudaMemcpyAsync(n.id, hid, np * 8, cudaMemcpyHostToDevice, ctx->s_in));
    ctx->id_bits_stale = true;                          // as in the whole-array branch: these may be other ids
    ++ctx->steps;
    for (int b = 0; b < kBatches; ++b) {
        const size_t p0 = (size_t)b * per;
        if (p0 >= np) break;
        const size_t cnt = std::min(per, np - p0);
        LP_CUDA(ctx, cudaMemcpyAsync(n.chi + p0 * nb, hchi + p0 * nb, cnt * nb * 8, cudaMemcpyHostToDevice, ctx->s_in));
        LP_CUDA(ctx, cudaEventRecord(ev_in[b], ctx->s_in));
        LP_CUDA(ctx, cudaStreamWaitEvent(s, ev_in[b], 0));
        if ((st = do_spectral(ctx, dt, io_in_place(ctx), true, s, (long long)p0, (long long)cnt)) != LP_OK) return st;
        LP_CUDA(ctx, cudaEventRecord(ev_k[b], s));
        LP_CUDA(ctx, cudaStreamWaitEvent(ctx->s_out, ev_k[b], 0));
        LP_CUDA(ctx, cudaMemcpyAsync(hchi + p0 * nb, n.chi + p0 * nb, cnt * nb * 8, cudaMemcpyDeviceToHost, ctx->s_out));
    }
    // positions are final once the last batch has run (s_out already waits for it); ids are unchanged
    LP_CUDA(ctx, cudaMemcpyAsync(hx, n.x, np * 8, cudaMemcpyDeviceToHost, ctx->s_out));
    LP_CUDA(ctx, cudaMemcpyAsync(hy, n.y, np * 8, cudaMemcpyDeviceToHost, ctx->s_out));
    LP_CUDA(ctx, cudaMemcpyAsync(hz, n.z, np * 8, cudaMemcpyDeviceToHost, ctx->s_out));
    LP_CUDA(ctx, cudaEventRecord(ev_done, ctx->s_out));
    LP_CUDA(ctx, cudaStreamWaitEvent(s, ev_done, 0));
    LP_CUDA(ctx, cudaStreamSynchronize(s));
    return LP_OK;
}

lp_status lp_get_diag(lp_ctx *ctx, lp_diag *out, void *stream)
{
    lp_status st = need_ready(ctx, false);
    if (st != LP_OK) return st;
    if (!out) return fail(ctx, LP_ERR_INVALID_ARG, "out is NULL");
    std::memset(out, 0, sizeof *out);
    out->np = ctx->cfg.np;
    out->steps = ctx->steps;
    out->sorts = ctx->sorts;
    if (ctx->cfg.np == 0) return LP_OK;
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    LpDiagDev *d = ctx->at<LpDiagDev>(ctx->lay.diag), h;
    LP_CUDA(ctx, cudaMemsetAsync(d, 0, sizeof(LpDiagDev), s));
    const bool have = ctx->spectra_done;
    // before the first spectral update n_sub / lost / status hold no data: reduce chi only
    if (!have) LP_CUDA(ctx, cudaMemsetAsync(ctx->at<int32_t>(ctx->lay.nsub), 0, (size_t)ctx->cfg.np * 4, s));
    st = count(ctx, lp_launch_diag(ctx->at<int32_t>(ctx->lay.nsub),
                                   (have && ctx->lost_user && !ctx->eng) ? ctx->at<double>(ctx->lay.lost) : nullptr,
                                   ctx->status_valid ? ctx->at<int32_t>(ctx->lay.status) : nullptr, ctx->now().chi, ctx->eng, ctx->tab,
                                   ctx->cfg.nbins, ctx->cfg.np, ctx->at<double>(ctx->lay.partial), d, s),
               "lp_diag_kernel launch");
    if (st != LP_OK) return st;
    LP_CUDA(ctx, cudaMemcpyAsync(&h, d, sizeof h, cudaMemcpyDeviceToHost, s));
    LP_CUDA(ctx, cudaStreamSynchronize(s));
    out->sum_substeps = h.sum_substeps;
    out->max_substeps = h.max_substeps;
    out->n_capped = h.n_capped;
    out->n_outside = h.n_outside;
    out->number = h.number;
    out->lost = h.lost;
    if (ctx->cap_is_error && h.n_capped > 0)        // (out is filled: the caller can still see how many)
        return fail(ctx, LP_ERR_UNSUPPORTED, "particles hit max_substeps in the last spectral update: their rows took "
                                             "substeps beyond the CFL bound (raise max_substeps or lower dt)");
    return LP_OK;
}

lp_status lp_set_cap_policy(lp_ctx *ctx, int error_on_cap)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    ctx->cap_is_error = error_on_cap != 0;
    return LP_OK;
}

lp_status lp_launch_count(const lp_ctx *ctx, int64_t *out)
{
    if (!ctx || !out) return LP_ERR_INVALID_ARG;
    *out = ctx->launches;
    return LP_OK;
}

lp_status lp_get_cfl_bins(const lp_ctx *ctx, int32_t *bins, int32_t *n)
{
    if (!ctx || !bins || !n) return LP_ERR_INVALID_ARG;
    *n = ctx->cand.n;
    for (int k = 0; k < ctx->cand.n; ++k) bins[k] = ctx->cand.bin[k];
    return LP_OK;
}

lp_status lp_timing_enable(lp_ctx *ctx, int max_records)
{
    if (!ctx || max_records < 0) return LP_ERR_INVALID_ARG;
    LP_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
    ctx->ev.clear();
    ctx->ev_used = 0;
    ctx->timing = max_records > 0;
    for (int i = 0; i < 2 * max_records; ++i) {
        cudaEvent_t e;
        LP_CUDA(ctx, cudaEventCreate(&e));
        ctx->ev.push_back(e);
    }
    return LP_OK;
}

lp_status lp_timing_read(lp_ctx *ctx, double *spectral_ms_sum, int32_t *n_records)
{
    if (!ctx || !spectral_ms_sum || !n_records) return LP_ERR_INVALID_ARG;
    double sum = 0.0;
    for (size_t i = 0; i + 1 < ctx->ev_used; i += 2) {
        LP_CUDA(ctx, cudaEventSynchronize(ctx->ev[i + 1]));
        float ms = 0.f;
        LP_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->ev[i], ctx->ev[i + 1]));
        sum += ms;
    }
    *spectral_ms_sum = sum;
    *n_records = (int32_t)(ctx->ev_used / 2);
    ctx->ev_used = 0;
    return LP_OK;
}

lp_status lp_get_bins(const lp_ctx *ctx, double *edges, double *widths)
{
    if (!ctx) return LP_ERR_INVALID_ARG;
    if (edges) std::memcpy(edges, ctx->h_edges.data(), ctx->h_edges.size() * sizeof(double));
    if (widths) std::memcpy(widths, ctx->h_widths.data(), ctx->h_widths.size() * sizeof(double));
    return LP_OK;
}

}  // extern "C"
