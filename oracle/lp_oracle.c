/*
 * oracle/lp_oracle.c -- CPU ORACLE for the Lagrangian-Particle (LP) hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_2602_23434_b200/ and neither imports the other.
 *
 * Plain, slow, scalar fp64 C.  Compile with  gcc -O2 -ffp-contract=off  so that no
 * a*b+c is fused: every + - * / sqrt floor below is one correctly rounded IEEE-754
 * operation, evaluated in the order written.  (The CUDA path reproduces the
 * key / gather / push arithmetic operation by operation so that indices and
 * positions can be compared bit for bit; reading R14.)
 *
 * What it computes, with the passage of /root/reference/PAPER.md each part follows
 * ("R<n>" = a reading listed in DESIGN.md section 3, taken where the paper is silent):
 *
 *   orc_bin_table        N_b log-spaced energy bins          PAPER.md:122, 282-284 (Eq. 13)      R1,R3
 *   orc_cell_key         containing cell of x_LP             PAPER.md:81-85 (sampling)           R15
 *   orc_sort_perm        order by (cell key, id)             not in the paper (north_star)       --
 *   orc_gather           trilinear sampling of v,B,rho       PAPER.md:85 ("sample fluid ...")    R2
 *   orc_push_stage0/1    two-stage predictor-corrector       PAPER.md:83 (Eq. 1), 218-227        R16
 *   orc_coefficients     gamma_g, dtau, c_r, a               PAPER.md:85, 96-99 (Eq. 4), 105-107 R4-R9
 *   orc_cfl_nsub         CFL-limited substep count           north_star                          R12
 *   orc_spectral_row     donor-cell upwind update of chi     PAPER.md:107 (Eq. 6)                R1,R10,R11
 *   orc_spectral_update  the three above for every particle  PAPER.md:218-231 (Particles_Spectra)
 *   orc_shock_row/update spectrum reset at a shock crossing  PAPER.md:110-122 (Eq. 7-8)          S1-S4
 *   orc_compact          deletion with hole filling          PAPER.md:190-199                    C1
 *   orc_push_rk3_stage   three-stage third-order pusher      PAPER.md:245, 258-260               K1
 *   orc_migrate_pack/unpack  exchange across rank interfaces PAPER.md:201-214                    M1-M3
 *   orc_moving_row/update    per-particle moving energy grid PAPER.md:107, 122, 606-613, 685     E1-E4
 *   orc_step             one whole step with frozen fields   PAPER.md:216-233 (Table 1)
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): brute-force cell search and O(N^2)
 * selection sort; constant / linear / cell-centre fields for the gather; uniform
 * flow, the closed form Eq. 10 and homologous flow for the pusher;
 * the analytic synchrotron-cooled power law, the adiabatic rho^{1/3} law, a
 * scale-invariance product formula, the loss steady state, number conservation,
 * positivity and hand-worked N_b = 2, 3 cases for the spectral update; hand-worked fractions, a closed
 * form and the paper's slope for the shock update; hand-worked cases and invariants for the compaction; the
 * cubic Taylor factor for the third-order pusher; a hand-worked two-rank case, the owner by brute force and
 * "everybody at home after three sweeps" for the exchange; hand-worked values, an independent ODE
 * integration, the synchrotron and rho^(1/3) laws and exact bin means of a cooled power law for the moving
 * energy grid.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t nx, ny, nz;        /* cells per axis; cell-centred data, index (k*ny + j)*nx + i   */
    double  xlo[3], xhi[3];    /* domain                                                         */
    int32_t periodic[3];       /* 1: periodic axis, 0: zero-gradient (clamped) axis              */
    int32_t nbins;             /* N_b                                                            */
    double  e_min, e_max;      /* outer bin edges                                                */
    double  kappa, u_rad;      /* c_r = kappa * (|B|^2/2 + u_rad)          (Eq. 4, R4-R6)        */
    double  cfl_e;             /* C_E, energy-space CFL number             (R12)                 */
    int32_t max_substeps;      /* cap on n_sub                             (R12)                 */
} orc_params;

/* ---------------------------------------------------------------- bins (R1, R3) */

/* N_b+1 log-spaced edges spanning exactly [e_min, e_max]; widths; geometric centres.
 * PAPER.md:122 defers the discretisation to [19]; Eq. 13 indexes
 * "N_b energy bins between e_min and e_max". */
void orc_bin_table(int32_t nbins, double e_min, double e_max,
                   double *E /*[nbins+1]*/, double *dE /*[nbins]*/, double *Ec /*[nbins]*/)
{
    for (int k = 0; k <= nbins; ++k)
        E[k] = e_min * pow(e_max / e_min, (double)k / (double)nbins);
    for (int i = 0; i < nbins; ++i) {
        dE[i] = E[i + 1] - E[i];
        Ec[i] = sqrt(E[i] * E[i + 1]);
    }
}

/* ---------------------------------------------------------------- cell key (R15) */

static int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* Containing cell per axis c = floor((x - xlo) * inv_dx), inv_dx = n / (xhi - xlo),
 * clamped to [0, n-1]; a face belongs to the upper cell.  key = (ck*ny + cj)*nx + ci. */
void orc_cell_key(const orc_params *g, int64_t np,
                  const double *x, const double *y, const double *z, uint32_t *key)
{
    const double idx = (double)g->nx / (g->xhi[0] - g->xlo[0]);
    const double idy = (double)g->ny / (g->xhi[1] - g->xlo[1]);
    const double idz = (double)g->nz / (g->xhi[2] - g->xlo[2]);
    for (int64_t p = 0; p < np; ++p) {
        int ci = clampi((int)floor((x[p] - g->xlo[0]) * idx), 0, g->nx - 1);
        int cj = clampi((int)floor((y[p] - g->xlo[1]) * idy), 0, g->ny - 1);
        int ck = clampi((int)floor((z[p] - g->xlo[2]) * idz), 0, g->nz - 1);
        key[p] = (uint32_t)((ck * g->ny + cj) * g->nx + ci);
    }
}

/* ---------------------------------------------------------------- sort */

typedef struct { uint32_t key; uint64_t id; int64_t src; } orc_sort_rec;

static int orc_cmp(const void *a, const void *b)
{
    const orc_sort_rec *p = (const orc_sort_rec *)a, *q = (const orc_sort_rec *)b;
    if (p->key != q->key) return p->key < q->key ? -1 : 1;
    if (p->id != q->id)   return p->id < q->id ? -1 : 1;
    return 0;
}

/* perm[n] = index (in the current order) of the particle that comes n-th when ordered
 * ascending by (key, id).  ids are unique, so the order is total and perm is unique. */
void orc_sort_perm(int64_t np, const uint32_t *key, const uint64_t *id, int64_t *perm)
{
    orc_sort_rec *r = (orc_sort_rec *)malloc((size_t)np * sizeof *r);
    for (int64_t p = 0; p < np; ++p) { r[p].key = key[p]; r[p].id = id[p]; r[p].src = p; }
    qsort(r, (size_t)np, sizeof *r, orc_cmp);
    for (int64_t p = 0; p < np; ++p) perm[p] = r[p].src;
    free(r);
}

/* ---------------------------------------------------------------- gather (R2) */

static int wrap_index(int i, int n, int periodic)
{
    if (periodic) { int m = i % n; return m < 0 ? m + n : m; }
    return clampi(i, 0, n - 1);
}

/* Trilinear interpolation of nq cell-centred fields at one position.
 * Per axis: s = (x - xlo)*inv_dx - 1/2, i0 = floor(s), f = s - i0; neighbours i0, i0+1
 * mapped by floor-mod (periodic) or clamped (zero gradient, as the outflow BC of
 * PAPER.md:276).  Corners are summed z outer, y, x inner; weight = (wz*wy)*wx. */
static void gather_point(const orc_params *g, int nq, const double *const *q,
                         double px, double py, double pz, double *out)
{
    const double idx = (double)g->nx / (g->xhi[0] - g->xlo[0]);
    const double idy = (double)g->ny / (g->xhi[1] - g->xlo[1]);
    const double idz = (double)g->nz / (g->xhi[2] - g->xlo[2]);
    double sx = (px - g->xlo[0]) * idx - 0.5, sy = (py - g->xlo[1]) * idy - 0.5,
           sz = (pz - g->xlo[2]) * idz - 0.5;
    double fx0 = floor(sx), fy0 = floor(sy), fz0 = floor(sz);
    double fx = sx - fx0, fy = sy - fy0, fz = sz - fz0;
    int i0 = (int)fx0, j0 = (int)fy0, k0 = (int)fz0;
    int ii[2] = { wrap_index(i0, g->nx, g->periodic[0]), wrap_index(i0 + 1, g->nx, g->periodic[0]) };
    int jj[2] = { wrap_index(j0, g->ny, g->periodic[1]), wrap_index(j0 + 1, g->ny, g->periodic[1]) };
    int kk[2] = { wrap_index(k0, g->nz, g->periodic[2]), wrap_index(k0 + 1, g->nz, g->periodic[2]) };
    double wx[2] = { 1.0 - fx, fx }, wy[2] = { 1.0 - fy, fy }, wz[2] = { 1.0 - fz, fz };
    for (int m = 0; m < nq; ++m) out[m] = 0.0;
    for (int cz = 0; cz < 2; ++cz)
        for (int cy = 0; cy < 2; ++cy)
            for (int cx = 0; cx < 2; ++cx) {
                double w = (wz[cz] * wy[cy]) * wx[cx];
                int64_t c = ((int64_t)kk[cz] * g->ny + jj[cy]) * g->nx + ii[cx];
                for (int m = 0; m < nq; ++m) out[m] = out[m] + w * q[m][c];
            }
}

/* out[m*np + p] = field m at particle p, m = 0..6 in the order vx,vy,vz,bx,by,bz,rho. */
void orc_gather(const orc_params *g, const double *const *fields7, int64_t np,
                const double *x, const double *y, const double *z, double *out7)
{
    for (int64_t p = 0; p < np; ++p) {
        double o[7];
        gather_point(g, 7, fields7, x[p], y[p], z[p], o);
        for (int m = 0; m < 7; ++m) out7[(int64_t)m * np + p] = o[m];
    }
}

/* ---------------------------------------------------------------- push (Eq. 1, R16) */

/* Stage 0 (Particles_RK#1): k1 = v(x^n), rho_old = rho(x^n),
 * x* = x^n + dt*k1.  x* is not wrapped (the gather wraps indices). */
void orc_push_stage0(const orc_params *g, const double *const *fields7, int64_t np,
                     const double *x, const double *y, const double *z, double dt,
                     double *k1 /*[3][np]*/, double *rho_old /*[np]*/, double *xs /*[3][np]*/,
                     int32_t nthreads)
{
    const double *q[4] = { fields7[0], fields7[1], fields7[2], fields7[6] };
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (int64_t p = 0; p < np; ++p) {
        double o[4];
        gather_point(g, 4, q, x[p], y[p], z[p], o);
        k1[p] = o[0]; k1[np + p] = o[1]; k1[2 * np + p] = o[2];
        rho_old[p] = o[3];
        xs[p]          = x[p] + dt * o[0];
        xs[np + p]     = y[p] + dt * o[1];
        xs[2 * np + p] = z[p] + dt * o[2];
    }
}

/* Periodic wrap into [lo, hi): x -= L*floor((x-lo)/L); a result >= hi becomes lo. */
static double wrap_pos(double x, double lo, double hi)
{
    double L = hi - lo;
    x = x - L * floor((x - lo) / L);
    if (x >= hi) x = lo;
    return x;
}

/* Stage 1 (Particles_RK#2 + Particles_Boundary): k2 = v(x*) from
 * the fields passed now (the caller may have advanced them);
 * x^{n+1} = x^n + (dt/2)*(k1 + k2)  (Heun).  Periodic axes are wrapped; on a
 * non-periodic axis the position is kept and bit (1 << axis) of status is set when
 * it lies outside [lo, hi). */
void orc_push_stage1(const orc_params *g, const double *const *fields7, int64_t np,
                     double *x, double *y, double *z, const double *xs, const double *k1,
                     double dt, int32_t *status /*[np] or NULL*/, int32_t nthreads)
{
    const double *q[3] = { fields7[0], fields7[1], fields7[2] };
    double *pos[3] = { x, y, z };
    const double hdt = 0.5 * dt;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (int64_t p = 0; p < np; ++p) {
        double k2[3];
        int32_t st = 0;
        gather_point(g, 3, q, xs[p], xs[np + p], xs[2 * np + p], k2);
        for (int d = 0; d < 3; ++d) {
            double xn = pos[d][p] + hdt * (k1[(int64_t)d * np + p] + k2[d]);
            if (g->periodic[d]) xn = wrap_pos(xn, g->xlo[d], g->xhi[d]);
            else if (xn < g->xlo[d] || xn >= g->xhi[d]) st |= (1 << d);
            pos[d][p] = xn;
        }
        if (status) status[p] = st;
    }
}

/* Third-order pusher (NEXT-4; PAPER.md:245, 258-260 show a "third order Runge-Kutta" next to the second
 * order one without naming the variant).  Reading K1: the three-stage Shu-Osher (SSP) scheme
 * that PLUTO's RK3 time stepping uses, one call per stage so that the caller can advance the fields in
 * between, as for the two-stage pusher:
 *   stage 0:  x0 = x^n (kept);  rho_old = rho(x^n);  x1 = x0 + dt v(x0)
 *   stage 1:  x2 = (3/4) x0 + (1/4) (x1 + dt v(x1))
 *   stage 2:  x^{n+1} = (x0 + 2 (x2 + dt v(x2))) / 3;  periodic wrap / outside flag as orc_push_stage1.
 * x, y, z hold the current stage position on entry and the next one on return; intermediate positions
 * are not wrapped (the gather wraps indices). */
void orc_push_rk3_stage(const orc_params *g, const double *const *fields7, int64_t np, int32_t stage,
                        double *x, double *y, double *z, double *x0 /*[3][np]*/, double dt,
                        double *rho_old /*[np], stage 0*/, int32_t *status /*[np] or NULL, stage 2*/)
{
    const double *q[4] = { fields7[0], fields7[1], fields7[2], fields7[6] };
    double *pos[3] = { x, y, z };
    for (int64_t p = 0; p < np; ++p) {
        double o[4];
        int32_t st = 0;
        gather_point(g, 4, q, x[p], y[p], z[p], o);
        for (int d = 0; d < 3; ++d) {
            const double cur = pos[d][p];
            const double adv = cur + dt * o[d];
            double xn;
            if (stage == 0) {
                x0[(int64_t)d * np + p] = cur;
                xn = adv;
            } else if (stage == 1) {
                xn = 0.75 * x0[(int64_t)d * np + p] + 0.25 * adv;
            } else {
                xn = (x0[(int64_t)d * np + p] + 2.0 * adv) / 3.0;
                if (g->periodic[d]) xn = wrap_pos(xn, g->xlo[d], g->xhi[d]);
                else if (xn < g->xlo[d] || xn >= g->xhi[d]) st |= (1 << d);
            }
            pos[d][p] = xn;
        }
        if (stage == 0 && rho_old) rho_old[p] = o[3];
        if (stage == 2 && status) status[p] = st;
    }
}

/* ---------------------------------------------------------------- coefficients (R4-R9) */

/* From v, B, rho_new gathered at x^{n+1} and rho_old gathered at x^n:
 *   gamma_g = 1/sqrt(1 - |v|^2)  (c = 1),  dtau = dt/gamma_g
 *   c_r     = kappa*(|B|^2/2 + u_rad)                                  PAPER.md:96-99 (Eq. 4)
 *   a       = -log(rho_new/rho_old)/(3 dtau)  = (1/3) div_mu u^mu      PAPER.md:105 (continuity), R7
 * so that d(eps)/d(tau) = -eps*(a + c_r*eps) is the bracket of Eq. 6. */
void orc_coefficients(const orc_params *g, double dt, const double v[3], const double B[3],
                      double rho_new, double rho_old, double *a, double *cr, double *dtau)
{
    double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    double b2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
    double gam = 1.0 / sqrt(1.0 - v2);
    *dtau = dt / gam;
    *cr = g->kappa * (0.5 * b2 + g->u_rad);
    *a = -log(rho_new / rho_old) / (3.0 * *dtau);
}

/* ---------------------------------------------------------------- CFL (R12) */

/* Edge velocities w_k = -E_k*(a + c_r*E_k); outflow rate of bin i is
 * (max(w_{i+1},0) - min(w_i,0))/dE_i; lambda = max over bins;
 * n_sub = max(1, ceil(dtau*lambda/C_E)), capped at max_substeps (return value's
 * sign is flipped when the cap was applied so that the caller can count it). */
int32_t orc_cfl_nsub(int32_t nbins, const double *E, const double *dE, double a, double cr,
                     double dtau, double cfl_e, int32_t max_substeps, double *lambda_out)
{
    double lam = 0.0;
    for (int i = 0; i < nbins; ++i) {
        double wl = -E[i] * (a + cr * E[i]);
        double wr = -E[i + 1] * (a + cr * E[i + 1]);
        double out = (fmax(wr, 0.0) - fmin(wl, 0.0)) / dE[i];
        if (out > lam) lam = out;
    }
    if (lambda_out) *lambda_out = lam;
    double need = ceil(dtau * lam / cfl_e);
    int32_t n = need < 1.0 ? 1 : (need > 2.0e9 ? 2000000000 : (int32_t)need);
    if (n > max_substeps) return -max_substeps;
    return n;
}

/* ---------------------------------------------------------------- substeps (Eq. 6, R1, R10, R11) */

/* n_sub explicit donor-cell steps of  d(chi)/d(tau) + d/d(eps)[w chi] = 0:
 *   F_k   = max(w_k,0)*chi_{k-1} + min(w_k,0)*chi_k      (interior edges)
 *   F_0   = min(w_0,0)*chi_0,  F_Nb = max(w_Nb,0)*chi_{Nb-1}   (no inflow, free outflow)
 *   chi_i <- chi_i - (dtau_s/dE_i)*(F_{i+1} - F_i),   dtau_s = dtau/n_sub
 * lost accumulates dtau_s*(F_Nb - F_0), the number that left through the ends. */
void orc_spectral_row(int32_t nbins, const double *E, const double *dE, double a, double cr,
                      double dtau, int32_t nsub, double *chi /*[nbins] in/out*/, double *lost)
{
    double *w = (double *)malloc((size_t)(nbins + 1) * sizeof(double));
    double *F = (double *)malloc((size_t)(nbins + 1) * sizeof(double));
    const double dts = dtau / (double)nsub;
    double lo = 0.0;
    for (int k = 0; k <= nbins; ++k) w[k] = -E[k] * (a + cr * E[k]);
    for (int s = 0; s < nsub; ++s) {
        F[0] = fmin(w[0], 0.0) * chi[0];
        for (int k = 1; k < nbins; ++k)
            F[k] = fmax(w[k], 0.0) * chi[k - 1] + fmin(w[k], 0.0) * chi[k];
        F[nbins] = fmax(w[nbins], 0.0) * chi[nbins - 1];
        for (int i = 0; i < nbins; ++i)
            chi[i] = chi[i] - (dts / dE[i]) * (F[i + 1] - F[i]);
        lo = lo + dts * (F[nbins] - F[0]);
    }
    if (lost) *lost = lo;
    free(w); free(F);
}

/* number of a row: sum_i chi_i dE_i  (diagnostic a10) */
double orc_row_number(int32_t nbins, const double *dE, const double *chi)
{
    double s = 0.0;
    for (int i = 0; i < nbins; ++i) s = s + chi[i] * dE[i];
    return s;
}

/* ---------------------------------------------------------------- shock crossing (Eq. 7-8; NEXT-1) */

/* Spectrum of a particle that crosses a shock of compression ratio r:
 *   chi_out(e) = C * Int_{e_min}^{e} chi_in(e') (e/e')^(-q+2) de'/e'            (Eq. 7)
 *              = C * e^(2-q) * Int_{e_min}^{e} chi_in(e') e'^(q-3) de',
 *   q = 3r/(r-1) + q_R                                                          (Eq. 8)
 * Readings (S1-S4): r is given per particle by the caller (the paper defines no
 * shock finder), r <= 1 means "no shock": the row is left untouched; q_R is a caller-supplied scalar;
 * the integral to the centre e_i of bin i is the midpoint sum over the bins below plus half of bin i,
 *   I_i = sum_{j<i} chi_j ec_j^(q-3) dE_j + (1/2) chi_i ec_i^(q-3) dE_i,   ec = geometric bin centre;
 * C ("a normalization that depends on the shock energy (see [19, 20])", not available here) keeps the
 * particle's number: sum_i chi_out_i dE_i = sum_i chi_in_i dE_i.  A row whose unnormalised result sums
 * to zero is left untouched.  Returns 1 if the row was changed. */
int32_t orc_shock_row(int32_t nbins, const double *E, const double *dE, double r, double q_r,
                      double *chi /*[nbins] in/out*/)
{
    if (!(r > 1.0)) return 0;
    const double q = 3.0 * r / (r - 1.0) + q_r;
    double *t = (double *)malloc((size_t)nbins * sizeof(double));
    double below = 0.0, n_in = 0.0, n_out = 0.0;
    for (int i = 0; i < nbins; ++i) {
        const double ec = sqrt(E[i] * E[i + 1]);
        const double term = chi[i] * pow(ec, q - 3.0) * dE[i];
        const double integral = below + 0.5 * term;
        t[i] = pow(ec, 2.0 - q) * integral;
        below = below + term;
        n_in = n_in + chi[i] * dE[i];
        n_out = n_out + t[i] * dE[i];
    }
    int32_t changed = 0;
    if (n_out != 0.0 && n_out == n_out) {
        const double c = n_in / n_out;
        for (int i = 0; i < nbins; ++i) chi[i] = c * t[i];
        changed = 1;
    }
    free(t);
    return changed;
}

/* every particle: row p with compression ratio r[p] */
void orc_shock_update(int32_t nbins, const double *E, const double *dE, int64_t np, const double *r,
                      double q_r, double *chi /*[np][nbins] in/out*/)
{
    for (int64_t p = 0; p < np; ++p) orc_shock_row(nbins, E, dE, r[p], q_r, chi + p * nbins);
}

/* the same with a per-particle energy grid (moving grid, readings E1-E4): row p is discretised on its own
 * edges eng[p][0..nbins], so its bin centres and widths are its own; orc_shock_row is written for any edges */
void orc_shock_update_grid(int32_t nbins, int64_t np, const double *eng /*[np][nbins+1]*/, const double *r,
                           double q_r, double *chi /*[np][nbins] in/out*/)
{
    double *dE = (double *)malloc((size_t)nbins * sizeof(double));
    for (int64_t p = 0; p < np; ++p) {
        const double *E = eng + p * (nbins + 1);
        for (int i = 0; i < nbins; ++i) dE[i] = E[i + 1] - E[i];
        orc_shock_row(nbins, E, dE, r[p], q_r, chi + p * nbins);
    }
    free(dE);
}

/* ---------------------------------------------------------------- deletion + hole filling (NEXT-2) */

/* The paper's compaction, step by step:
 *  1. flag and count the N_del particles to delete;  2. save the indices i_del of the flagged particles that
 *  lie below N_p - N_del (the holes);  3. collect the indices i_f of the fillers, the particles stored at
 *  i >= N_p - N_del that are not deleted;  4. copy every parameter of the fillers into the holes;
 *  5. shrink to N_p - N_del.
 * Reading (C1): the paper does not say which filler goes into which hole; here the k-th hole in
 * ascending index order receives the k-th filler in ascending index order.  The surviving set is unique,
 * the arrangement follows from this pairing.  Returns the new particle count. */
int64_t orc_compact(int64_t np, const int32_t *flag, int32_t nbins,
                    double *x, double *y, double *z, uint64_t *id, double *chi /*[np][nbins]*/)
{
    int64_t ndel = 0;
    for (int64_t i = 0; i < np; ++i) if (flag[i]) ++ndel;                         /* step 1 */
    const int64_t keep = np - ndel;
    int64_t *holes = (int64_t *)malloc((size_t)(np > 0 ? np : 1) * sizeof(int64_t));
    int64_t *fill = (int64_t *)malloc((size_t)(np > 0 ? np : 1) * sizeof(int64_t));
    int64_t nh = 0, nf = 0;
    for (int64_t i = 0; i < keep; ++i) if (flag[i]) holes[nh++] = i;              /* step 2 */
    for (int64_t i = keep; i < np; ++i) if (!flag[i]) fill[nf++] = i;             /* step 3 */
    for (int64_t k = 0; k < nh && k < nf; ++k) {                                  /* step 4 */
        const int64_t d = holes[k], s = fill[k];
        x[d] = x[s]; y[d] = y[s]; z[d] = z[s]; id[d] = id[s];
        for (int32_t b = 0; b < nbins; ++b) chi[d * nbins + b] = chi[s * nbins + b];
    }
    free(holes); free(fill);
    return keep;                                                                  /* step 5 */
}

/* ---------------------------------------------------------------- particle migration (NEXT-3) */

/* Exchange of the particles that crossed an inter-rank interface, one direction at a
 * time ("three steps for the three parallel directions"), a left and a right neighbour per direction.
 * The paper's eight steps, as seen by ONE rank that owns [lo, hi) along `axis`:
 *   1. collect holes (the leavers) and count how many particles go to each neighbour
 *   2.-3. (receive posted, buffers sized: the caller's business)
 *   4. pack the leavers into the two send buffers
 *   5.-7. (send, resize the container, wait)
 *   8. copy the arrivals into the holes left by the leavers and compact.
 * Readings (M1-M3; the paper gives the steps, not these details):
 *  M1 where a particle goes.  Positions were wrapped into the global box [glo, ghi) by the pusher
 *     (Particles_Boundary precedes Particles_Exchange), so a particle that left through
 *     the low face of the first rank of a periodic axis sits near ghi.  A particle outside [lo, hi) goes to
 *     the neighbour through whose face the shorter way leads, the other way being the one around the
 *     periodic box:  x < lo:  left over lo - x,  right over (x + L) - hi;   x >= hi:  right over x - hi,
 *     left over lo - (x - L);  L = ghi - glo.  A tie, or a non-periodic axis, takes the plain side.
 *  M2 order inside a send buffer: ascending index of the leavers.
 *  M3 where arrivals go: the arrivals from the left, then those from the right, in buffer order; the k-th
 *     arrival goes into the k-th hole (ascending index); arrivals beyond the holes are appended behind the
 *     last particle; holes beyond the arrivals are closed by the compaction of Section 3.2 (orc_compact,
 *     reading C1) with exactly those holes flagged. */
int32_t orc_migrate_dest(double x, double lo, double hi, double glo, double ghi, int32_t periodic)
{
    if (x >= lo && x < hi) return 0;
    const double L = ghi - glo;
    if (x < lo) {
        if (periodic) {
            const double left = lo - x, right = (x + L) - hi;
            if (right >= 0.0 && right < left) return 2;
        }
        return 1;
    }
    if (periodic) {
        const double right = x - hi, left = lo - (x - L);
        if (left >= 0.0 && left < right) return 1;
    }
    return 2;      /* x >= hi (or NaN) */
}

/* Steps 1 and 4.  dest[p] in {0, 1, 2}; holes[] = the leavers' indices ascending (n_left + n_right of
 * them); the leavers' parameters are copied, in ascending index order, into the left buffer
 * (lx, ly, lz, lid, lchi[.][nbins]) and the right buffer (r...), each with room for np particles. */
void orc_migrate_pack(int64_t np, int32_t nbins, int32_t axis, double lo, double hi, double glo, double ghi,
                      int32_t periodic, const double *x, const double *y, const double *z, const uint64_t *id,
                      const double *chi, int32_t *dest, int64_t *holes, int64_t *n_left, int64_t *n_right,
                      double *lx, double *ly, double *lz, uint64_t *lid, double *lchi,
                      double *rx, double *ry, double *rz, uint64_t *rid, double *rchi)
{
    const double *pos = axis == 0 ? x : (axis == 1 ? y : z);
    int64_t nl = 0, nr = 0, nh = 0;
    for (int64_t p = 0; p < np; ++p) {                                           /* step 1 */
        dest[p] = orc_migrate_dest(pos[p], lo, hi, glo, ghi, periodic);
        if (dest[p]) holes[nh++] = p;
    }
    for (int64_t p = 0; p < np; ++p) {                                           /* step 4 */
        if (dest[p] == 1) {
            lx[nl] = x[p]; ly[nl] = y[p]; lz[nl] = z[p]; lid[nl] = id[p];
            for (int32_t b = 0; b < nbins; ++b) lchi[nl * nbins + b] = chi[p * nbins + b];
            ++nl;
        } else if (dest[p] == 2) {
            rx[nr] = x[p]; ry[nr] = y[p]; rz[nr] = z[p]; rid[nr] = id[p];
            for (int32_t b = 0; b < nbins; ++b) rchi[nr * nbins + b] = chi[p * nbins + b];
            ++nr;
        }
    }
    *n_left = nl; *n_right = nr;
}

/* Step 8.  The arrays have room for np + n_from_left + n_from_right particles.  Returns the new count. */
int64_t orc_migrate_unpack(int64_t np, int32_t nbins, const int64_t *holes, int64_t nholes,
                           int64_t n_from_left, const double *lx, const double *ly, const double *lz,
                           const uint64_t *lid, const double *lchi,
                           int64_t n_from_right, const double *rx, const double *ry, const double *rz,
                           const uint64_t *rid, const double *rchi,
                           double *x, double *y, double *z, uint64_t *id, double *chi)
{
    const int64_t nin = n_from_left + n_from_right;
    int64_t count = np;
    for (int64_t k = 0; k < nin; ++k) {
        const int from_right = k >= n_from_left;
        const int64_t s = from_right ? k - n_from_left : k;
        const int64_t d = k < nholes ? holes[k] : count++;                       /* hole, else appended */
        x[d] = from_right ? rx[s] : lx[s];
        y[d] = from_right ? ry[s] : ly[s];
        z[d] = from_right ? rz[s] : lz[s];
        id[d] = from_right ? rid[s] : lid[s];
        for (int32_t b = 0; b < nbins; ++b) chi[d * nbins + b] = from_right ? rchi[s * nbins + b] : lchi[s * nbins + b];
    }
    if (nin < nholes) {                                                          /* compact the rest away */
        int32_t *flag = (int32_t *)calloc((size_t)(np > 0 ? np : 1), sizeof(int32_t));
        for (int64_t k = nin; k < nholes; ++k) flag[holes[k]] = 1;
        count = orc_compact(np, flag, nbins, x, y, z, id, chi);
        free(flag);
    }
    return count;
}

/* ---------------------------------------------------------------- moving energy grid (NEXT-5) */

/* Listing 3 gives every particle its own energy array eng_ next to chi_ and the text
 * defers the method to Section 2.3.2 of [19], which is not available.  Readings (DESIGN.md
 * section 3, E1-E4):
 *  E1 eng holds the particle's N_b + 1 bin edges, chi_i the mean of chi over [eng_i, eng_{i+1}].
 *  E2 over one step the edges follow the characteristics of Eq. 6,
 *       d(eps)/d(tau) = -eps (a + c_r eps),      a, c_r as orc_coefficients, frozen over the step (R9),
 *     whose solution over dtau is, with s = a dtau:
 *       eps(dtau) = eps0 e^{-s} / (1 + beta eps0),   beta = c_r dtau (1 - e^{-s}) / s   (= c_r dtau for s = 0).
 *     (e^{-s} = (rho_new/rho_old)^{1/3}: the adiabatic law; a = 0: eps0 / (1 + c_r eps0 dtau), the
 *     synchrotron law of north_star.)
 *  E3 Eq. 6 is a conservation law, so the number of a bin moves with its edges:
 *       chi_i <- chi_i (eng_{i+1} - eng_i)_old / (eng_{i+1} - eng_i)_new.
 *     No flux crosses an edge: no CFL limit, no substeps, nothing is lost through the ends.
 *  E4 the grid starts as the fixed log-spaced table (orc_bin_table). */
void orc_moving_row(int32_t nbins, double a, double cr, double dtau,
                    double *eng /*[nbins+1] in/out*/, double *chi /*[nbins] in/out*/)
{
    const double s = a * dtau;
    const double alpha = exp(-s);
    const double beta = (s != 0.0) ? cr * dtau * (-expm1(-s) / s) : cr * dtau;
    double *en = (double *)malloc((size_t)(nbins + 1) * sizeof(double));
    for (int k = 0; k <= nbins; ++k) en[k] = eng[k] * alpha / (1.0 + beta * eng[k]);
    for (int i = 0; i < nbins; ++i) chi[i] = chi[i] * (eng[i + 1] - eng[i]) / (en[i + 1] - en[i]);
    for (int k = 0; k <= nbins; ++k) eng[k] = en[k];
    free(en);
}

/* Particles_Spectra with the moving grid: gather at the current position, coefficients, orc_moving_row. */
void orc_moving_update(const orc_params *g, const double *const *fields7, int64_t np,
                       const double *x, const double *y, const double *z, const double *rho_old, double dt,
                       double *eng /*[np][nbins+1]*/, double *chi /*[np][nbins]*/, int32_t nthreads)
{
    const int nb = g->nbins;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (int64_t p = 0; p < np; ++p) {
        double o[7], a, cr, dtau;
        gather_point(g, 7, fields7, x[p], y[p], z[p], o);
        orc_coefficients(g, dt, &o[0], &o[3], o[6], rho_old[p], &a, &cr, &dtau);
        orc_moving_row(nb, a, cr, dtau, eng + p * (nb + 1), chi + p * nb);
    }
}

/* ---------------------------------------------------------------- whole update / step */

/* Particles_Spectra: for every particle, gather v,B,rho at the
 * current position from the current fields, form the coefficients, the substep count
 * and run the substeps on its row chi[p*nbins .. ].  nsub_out gets n_sub (negative if
 * capped), lost_out the number lost this call.  nthreads > 1 splits the particle loop
 * with OpenMP (here and in the two push stages); the arithmetic per particle is unchanged. */
void orc_spectral_update(const orc_params *g, const double *const *fields7, int64_t np,
                         const double *x, const double *y, const double *z,
                         const double *rho_old, double dt, double *chi /*[np][nbins]*/,
                         int32_t *nsub_out /*or NULL*/, double *lost_out /*or NULL*/,
                         int32_t nthreads)
{
    const int nb = g->nbins;
    double *E = (double *)malloc((size_t)(nb + 1) * sizeof(double));
    double *dE = (double *)malloc((size_t)nb * sizeof(double));
    double *Ec = (double *)malloc((size_t)nb * sizeof(double));
    orc_bin_table(nb, g->e_min, g->e_max, E, dE, Ec);
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (int64_t p = 0; p < np; ++p) {
        double o[7], a, cr, dtau, lost;
        gather_point(g, 7, fields7, x[p], y[p], z[p], o);
        orc_coefficients(g, dt, &o[0], &o[3], o[6], rho_old[p], &a, &cr, &dtau);
        int32_t n = orc_cfl_nsub(nb, E, dE, a, cr, dtau, g->cfl_e, g->max_substeps, NULL);
        orc_spectral_row(nb, E, dE, a, cr, dtau, n < 0 ? -n : n, chi + p * nb, &lost);
        if (nsub_out) nsub_out[p] = n;
        if (lost_out) lost_out[p] = lost;
    }
    free(E); free(dE); free(Ec);
}

/* One step with frozen fields (the build's lp_step): stage 0, stage 1 + wrap,
 * spectral update at x^{n+1} with rho_old from stage 0.  Order of Table 1
 * with the fluid stages removed. */
void orc_step(const orc_params *g, const double *const *fields7, int64_t np,
              double *x, double *y, double *z, double dt, double *chi,
              int32_t *nsub_out, double *lost_out, int32_t *status, int32_t nthreads)
{
    double *k1 = (double *)malloc((size_t)np * 3 * sizeof(double));
    double *xs = (double *)malloc((size_t)np * 3 * sizeof(double));
    double *rho_old = (double *)malloc((size_t)np * sizeof(double));
    orc_push_stage0(g, fields7, np, x, y, z, dt, k1, rho_old, xs, nthreads);
    orc_push_stage1(g, fields7, np, x, y, z, xs, k1, dt, status, nthreads);
    orc_spectral_update(g, fields7, np, x, y, z, rho_old, dt, chi, nsub_out, lost_out, nthreads);
    free(k1); free(xs); free(rho_old);
}
