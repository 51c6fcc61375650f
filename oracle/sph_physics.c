/* ORACLE B - physics.  TEST INFRASTRUCTURE ONLY (tests/, __graft_entry__.smoke(),
 * bench.py cpu_baseline / --impl reference).  Never linked, imported or called by the
 * product path; shares no code, header, table or constant with the CUDA path.
 *
 * Plain, slow, fp64, gather-form implementation of the SPH equations of
 * arXiv 1210.1017 (line numbers are /root/reference/PAPER.md):
 *
 *   continuity   d rho_i/dt = sum_j m_j v_ij . grad_i W_ij                       Eq. (7)  L101
 *   momentum     d v_i /dt  = - sum_j m_j (p_i/rho_i^2 + p_j/rho_j^2 + Pi_ij)
 *                              grad_i W_ij + g                                   Eq. (9)  L106
 *                (the extracted text prints p/rho; the dimensionally consistent p/rho^2
 *                 form is the reading taken - DESIGN.md reading A2 - and it is pinned by
 *                 the linear-pressure-field test)
 *   viscosity    Pi_ij = -alpha cbar_ij mu_ij / rhobar_ij  if r_ij.v_ij < 0, else 0,
 *                mu_ij = h v_ij.r_ij / (r_ij^2 + eta^2), eta = 0.1 h                      L112
 *   state        p = B[(rho/rho0)^gamma - 1],  B = c0^2 rho0 / gamma, gamma = 7           L112
 *   sound speed  c_i = sqrt(dp/drho)|rho_i = c0 (rho_i/rho0)^((gamma-1)/2)   (reading A3) L112
 *   kernel       compact support 2h (kappa = 2), L77, L81.  kernel = 0: Wendland C2 (the
 *                kernel BASELINE.json binds); kernel = 1: cubic spline (the paper's, L81).
 *   boundaries   dynamic boundary particles obey the same equations but position and
 *                velocity are not integrated (L116): their acceleration is defined 0.
 *   neighbours   "all other particles within its support domain of 2h" (L132): j != i,
 *                0 < |r_ij| < 2h.  mode 0 = brute force O(N^2); mode 1 = own cell list of
 *                2h cells (L140, L146).  Both sum the accepted neighbours in ascending-id
 *                order, so they agree bit for bit.
 *   integrator   second-order Verlet (L150); formulas are reading A7.
 *
 * Optional periodic box (minimum image) exists ONLY here, for the momentum pin.
 *
 *   time step    variable dt of reading A8b (orc_time_step below; L150, L222).
 *
 * Pins: tests/test_oracle_physics.py (time step: two-particle hand values, lattice expansion,
 * per-slab minimum, numpy brute force; kernel integral, gradient vs finite difference,
 * EOS slope, divergence/pressure-gradient consistency, two-particle closed forms, pair
 * antisymmetry, brute force vs cell list, free fall, hydrostatic column).
 * Unpinned: absolute dam-break trajectories (the paper prints none) - "parity unpinned".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double h, rho0, c0, alpha, gamma;
    double g[3];
    double mass_fluid, mass_bound;
    int kernel;          /* 0 Wendland C2, 1 cubic spline */
    int periodic[3];
    double box_min[3], box_len[3];
} orc_params;

static const double PI = 3.14159265358979323846;

int orc_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* W(r) */
double orc_W(const orc_params *P, double r)
{
    double h = P->h, q = r / h;
    if (q >= 2.0) return 0.0;
    if (P->kernel == 0) {
        double aD = 21.0 / (16.0 * PI * h * h * h);
        double t = 1.0 - 0.5 * q;
        return aD * t * t * t * t * (2.0 * q + 1.0);
    } else {
        double aD = 1.0 / (PI * h * h * h);
        if (q <= 1.0) return aD * (1.0 - 1.5 * q * q + 0.75 * q * q * q);
        double t = 2.0 - q;
        return aD * 0.25 * t * t * t;
    }
}

/* F(r) = (dW/dr)/r, so that grad_i W_ij = F(|r_ij|) r_ij */
double orc_F(const orc_params *P, double r)
{
    double h = P->h, q = r / h;
    if (q >= 2.0) return 0.0;
    if (P->kernel == 0) {
        double aD = 21.0 / (16.0 * PI * h * h * h);
        double t = 1.0 - 0.5 * q;
        return -5.0 * aD * t * t * t / (h * h);
    } else {
        double aD = 1.0 / (PI * h * h * h);
        double dWdq;
        if (q <= 1.0) dWdq = aD * (-3.0 * q + 2.25 * q * q);
        else { double t = 2.0 - q; dWdq = -0.75 * aD * t * t; }
        return dWdq / (h * r);
    }
}

double orc_pressure(const orc_params *P, double rho)
{
    double B = P->c0 * P->c0 * P->rho0 / P->gamma;
    return B * (pow(rho / P->rho0, P->gamma) - 1.0);
}

double orc_sound_speed(const orc_params *P, double rho)
{
    return P->c0 * pow(rho / P->rho0, 0.5 * (P->gamma - 1.0));
}

static inline void rij_of(const orc_params *P, const double *ri, const double *rj, double *d)
{
    for (int k = 0; k < 3; ++k) {
        d[k] = ri[k] - rj[k];
        if (P->periodic[k]) d[k] -= P->box_len[k] * nearbyint(d[k] / P->box_len[k]);
    }
}

/* contribution of neighbour j to particle i; returns 1 if j is a neighbour */
static inline int pair(const orc_params *P, int fluid_i,
                       const double *ri, const double *vi, double rhoi, double pi_, double ci,
                       const double *rj, const double *vj, double rhoj, double pj, double cj,
                       double mj, double *acc, double *drho)
{
    double d[3];
    rij_of(P, ri, rj, d);
    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    double h = P->h;
    if (!(r2 < 4.0 * h * h) || !(r2 > 0.0)) return 0;
    double r = sqrt(r2);
    double F = orc_F(P, r);
    double dv[3] = { vi[0] - vj[0], vi[1] - vj[1], vi[2] - vj[2] };
    double dot = dv[0] * d[0] + dv[1] * d[1] + dv[2] * d[2];
    *drho += mj * dot * F;                                  /* Eq. (7) */
    if (fluid_i) {
        double Pi = 0.0;
        if (dot < 0.0) {                                    /* L112 */
            double eta2 = 0.01 * h * h;
            double mu = h * dot / (r2 + eta2);
            double cbar = 0.5 * (ci + cj);
            double rhobar = 0.5 * (rhoi + rhoj);
            Pi = -P->alpha * cbar * mu / rhobar;
        }
        double coef = -mj * (pi_ / (rhoi * rhoi) + pj / (rhoj * rhoj) + Pi) * F;   /* Eq. (9) */
        acc[0] += coef * d[0];
        acc[1] += coef * d[1];
        acc[2] += coef * d[2];
    }
    return 1;
}

static int cmp_long(const void *a, const void *b)
{
    long x = *(const long *)a, y = *(const long *)b;
    return (x > y) - (x < y);
}

/* Right-hand sides of Eqs. (7) and (9) for every particle.
 * r, v: n*3; rho, type: n; p_override: NULL, or n prescribed pressures (bypasses the EOS;
 * used by the linear-pressure-field pin).  mode 0 brute force, 1 cell list.
 * acc: n*3 (boundary particles: 0), drho: n.  Returns 0, or -1 on bad arguments. */
int orc_rates(const orc_params *P, long n, const double *r, const double *v, const double *rho,
              const unsigned char *type, const double *p_override, int mode,
              double *acc, double *drho)
{
    if (n < 0 || P->h <= 0.0) return -1;
    double *p = (double *)malloc(sizeof(double) * (n > 0 ? n : 1));
    double *c = (double *)malloc(sizeof(double) * (n > 0 ? n : 1));
    for (long i = 0; i < n; ++i) {
        p[i] = p_override ? p_override[i] : orc_pressure(P, rho[i]);
        c[i] = orc_sound_speed(P, rho[i]);
    }
    double cs = 2.0 * P->h;
    long nc[3] = { 1, 1, 1 };
    double lo[3] = { 0, 0, 0 };
    long *cell_start = NULL, *cell_items = NULL, *cell_of = NULL;
    if (mode == 1 && n > 0) {
        for (int k = 0; k < 3; ++k) {
            if (P->periodic[k]) {
                lo[k] = P->box_min[k];
                nc[k] = (long)floor(P->box_len[k] / cs);
                if (nc[k] < 3) { mode = 0; }
            } else {
                double mn = r[k], mx = r[k];
                for (long i = 1; i < n; ++i) { double x = r[3 * i + k]; if (x < mn) mn = x; if (x > mx) mx = x; }
                lo[k] = mn;
                nc[k] = (long)floor((mx - mn) / cs) + 1;
            }
        }
    }
    if (mode == 1 && n > 0) {
        long ncells = nc[0] * nc[1] * nc[2];
        cell_start = (long *)calloc((size_t)ncells + 1, sizeof(long));
        cell_items = (long *)malloc(sizeof(long) * n);
        cell_of = (long *)malloc(sizeof(long) * n);
        for (long i = 0; i < n; ++i) {
            long cc[3];
            for (int k = 0; k < 3; ++k) {
                double x = r[3 * i + k];
                double w = P->periodic[k] ? P->box_len[k] / (double)nc[k] : cs;
                if (P->periodic[k]) x -= P->box_len[k] * floor((x - lo[k]) / P->box_len[k]);
                long ck = (long)floor((x - lo[k]) / w);
                if (ck < 0) ck = 0;
                if (ck > nc[k] - 1) ck = nc[k] - 1;
                cc[k] = ck;
            }
            cell_of[i] = (cc[0] * nc[1] + cc[1]) * nc[2] + cc[2];
            cell_start[cell_of[i] + 1]++;
        }
        for (long cidx = 0; cidx < ncells; ++cidx) cell_start[cidx + 1] += cell_start[cidx];
        long *fill = (long *)malloc(sizeof(long) * ncells);
        memcpy(fill, cell_start, sizeof(long) * ncells);
        for (long i = 0; i < n; ++i) cell_items[fill[cell_of[i]]++] = i;
        free(fill);
    }

#pragma omp parallel
    {
        long cap = 256, *nb = (long *)malloc(sizeof(long) * cap);
#pragma omp for schedule(dynamic, 64)
        for (long i = 0; i < n; ++i) {
            double a[3] = { 0, 0, 0 }, dr = 0.0;
            int fl = (type[i] == 0);
            if (mode == 0) {
                for (long j = 0; j < n; ++j) {
                    if (j == i) continue;
                    double mj = type[j] == 0 ? P->mass_fluid : P->mass_bound;
                    pair(P, fl, r + 3 * i, v + 3 * i, rho[i], p[i], c[i],
                         r + 3 * j, v + 3 * j, rho[j], p[j], c[j], mj, a, &dr);
                }
            } else {
                /* candidates from the 27 cells around i's cell (L146), then ascending id */
                long ci_ = cell_of[i];
                long cz = ci_ % nc[2], cy = (ci_ / nc[2]) % nc[1], cx = ci_ / (nc[2] * nc[1]);
                long cnt = 0;
                long seen[27]; int nseen = 0;
                for (long dx = -1; dx <= 1; ++dx)
                for (long dy = -1; dy <= 1; ++dy)
                for (long dz = -1; dz <= 1; ++dz) {
                    long c3[3] = { cx + dx, cy + dy, cz + dz };
                    int ok = 1;
                    for (int k = 0; k < 3; ++k) {
                        if (P->periodic[k]) c3[k] = (c3[k] + nc[k]) % nc[k];
                        else if (c3[k] < 0 || c3[k] >= nc[k]) ok = 0;
                    }
                    if (!ok) continue;
                    long cidx = (c3[0] * nc[1] + c3[1]) * nc[2] + c3[2];
                    int dup = 0;
                    for (int s = 0; s < nseen; ++s) if (seen[s] == cidx) dup = 1;
                    if (dup) continue;
                    seen[nseen++] = cidx;
                    for (long s = cell_start[cidx]; s < cell_start[cidx + 1]; ++s) {
                        long j = cell_items[s];
                        if (j == i) continue;
                        double d[3];
                        rij_of(P, r + 3 * i, r + 3 * j, d);
                        double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                        if (!(r2 < 4.0 * P->h * P->h) || !(r2 > 0.0)) continue;
                        if (cnt == cap) { cap *= 2; nb = (long *)realloc(nb, sizeof(long) * cap); }
                        nb[cnt++] = j;
                    }
                }
                qsort(nb, (size_t)cnt, sizeof(long), cmp_long);
                for (long s = 0; s < cnt; ++s) {
                    long j = nb[s];
                    double mj = type[j] == 0 ? P->mass_fluid : P->mass_bound;
                    pair(P, fl, r + 3 * i, v + 3 * i, rho[i], p[i], c[i],
                         r + 3 * j, v + 3 * j, rho[j], p[j], c[j], mj, a, &dr);
                }
            }
            if (fl) { a[0] += P->g[0]; a[1] += P->g[1]; a[2] += P->g[2]; }
            else { a[0] = a[1] = a[2] = 0.0; }
            acc[3 * i] = a[0]; acc[3 * i + 1] = a[1]; acc[3 * i + 2] = a[2];
            drho[i] = dr;
        }
        free(nb);
    }
    free(p); free(c);
    free(cell_start); free(cell_items); free(cell_of);
    return 0;
}

/* Variable time step (L150: "The size of the integration time step varies throughout each
 * simulation according to the Courant-Friedrichs-Lewy (CFL) condition [20] and the magnitude of
 * the interactions.  Here, minimum and maximum values of certain physical quantities need to be
 * found among all particles"; L222: every sub-domain k determines its own dt_k, the step uses the
 * minimum).  The paper gives no formula; reading A8b takes the usual pair of limits,
 *     dt_f  = sqrt(h / max_i |a_i|)                    over fluid particles   ("magnitude of the interactions")
 *     dt_cv = h / max_i (c_i + max_j |mu_ij|)          over all particles     (CFL with the viscous signal speed)
 *     dt    = cfl * min(dt_f, dt_cv),
 * mu_ij = h v_ij.r_ij / (r_ij^2 + eta^2) as in L112, j over the neighbours 0 < r_ij < cut * 2h.
 * |mu_ij| does not vanish at the edge of the support, so max_j is discontinuous in the cut-off:
 * `cut` (1 for the definition) lets a test bracket an fp32 implementation between cut = 1 -+ eps.
 * Brute force O(N^2).  slab_of: NULL, or the owning sub-domain of every particle; then
 * amax_slab / smax_slab (n_slabs each) receive the per-sub-domain maxima of |a| and c + mu.
 * mu_out: NULL or n (max_j |mu_ij| per particle). */
int orc_time_step(const orc_params *P, long n, const double *r, const double *v, const double *rho,
                  const unsigned char *type, const double *acc, double cfl, double cut,
                  const long *slab_of, int n_slabs, double *amax_slab, double *smax_slab,
                  double *mu_out, double *dt_out /* dt, dt_f, dt_cv */)
{
    if (!P || n < 0 || !dt_out) return -1;
    double h = P->h, eta2 = 0.01 * h * h, rc2 = 4.0 * h * h * cut * cut;
    double *mu = (double *)calloc(n > 0 ? n : 1, sizeof(double));
    if (!mu) return -1;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) {
        double m = 0.0;
        for (long j = 0; j < n; ++j) {
            if (j == i) continue;
            double d[3];
            rij_of(P, r + 3 * i, r + 3 * j, d);
            double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            if (!(r2 < rc2) || !(r2 > 0.0)) continue;
            double dot = (v[3 * i] - v[3 * j]) * d[0] + (v[3 * i + 1] - v[3 * j + 1]) * d[1] +
                         (v[3 * i + 2] - v[3 * j + 2]) * d[2];
            double a = fabs(h * dot / (r2 + eta2));
            if (a > m) m = a;
        }
        mu[i] = m;
    }
    double amax = 0.0, smax = 0.0;
    for (int k = 0; k < n_slabs; ++k) { if (amax_slab) amax_slab[k] = 0.0; if (smax_slab) smax_slab[k] = 0.0; }
    for (long i = 0; i < n; ++i) {
        double s = orc_sound_speed(P, rho[i]) + mu[i];
        if (s > smax) smax = s;
        double a = 0.0;
        if (!type || type[i] == 0) {
            a = sqrt(acc[3 * i] * acc[3 * i] + acc[3 * i + 1] * acc[3 * i + 1] + acc[3 * i + 2] * acc[3 * i + 2]);
            if (a > amax) amax = a;
        }
        if (slab_of && n_slabs > 0) {
            long k = slab_of[i];
            if (k >= 0 && k < n_slabs) {
                if (smax_slab && s > smax_slab[k]) smax_slab[k] = s;
                if (amax_slab && a > amax_slab[k]) amax_slab[k] = a;
            }
        }
        if (mu_out) mu_out[i] = mu[i];
    }
    free(mu);
    double dt_f = amax > 0.0 ? sqrt(h / amax) : INFINITY;
    double dt_cv = smax > 0.0 ? h / smax : INFINITY;
    dt_out[1] = dt_f;
    dt_out[2] = dt_cv;
    dt_out[0] = cfl * (dt_f < dt_cv ? dt_f : dt_cv);
    return 0;
}

/* Number of neighbours (0 < r < 2h) of each particle by brute force; used by structure
 * pins (halo sufficiency).  nbr_count: n. */
int orc_neighbour_pairs(const orc_params *P, long n, const double *r, long max_pairs,
                        long *pairs_out /* 2*max_pairs */, long *n_pairs)
{
    long cnt = 0;
    for (long i = 0; i < n; ++i)
        for (long j = 0; j < n; ++j) {
            if (i == j) continue;
            double d[3];
            rij_of(P, r + 3 * i, r + 3 * j, d);
            double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            if (r2 < 4.0 * P->h * P->h && r2 > 0.0) {
                if (cnt < max_pairs) { pairs_out[2 * cnt] = i; pairs_out[2 * cnt + 1] = j; }
                cnt++;
            }
        }
    *n_pairs = cnt;
    return cnt <= max_pairs ? 0 : -1;
}

/* Second-order Verlet update (L150; reading A7):
 *   corrective step (every Ns-th step and step 0):  v+ = v + dt a,      rho+ = rho + dt drho
 *   otherwise:                                       v+ = v_m1 + 2dt a,  rho+ = rho_m1 + 2dt drho
 *   always                                           r+ = r + dt v + dt^2 a / 2
 *   then (v_m1, rho_m1) <- (v, rho).  Boundary particles: density lines only (L116). */
void orc_verlet(long n, double *r, double *v, double *rho, double *v_m1, double *rho_m1,
                const unsigned char *type, const double *acc, const double *drho,
                double dt, int corrective)
{
    for (long i = 0; i < n; ++i) {
        double rho_new = corrective ? rho[i] + dt * drho[i] : rho_m1[i] + 2.0 * dt * drho[i];
        if (type[i] == 0) {
            for (int k = 0; k < 3; ++k) {
                double vk = v[3 * i + k], ak = acc[3 * i + k];
                double v_new = corrective ? vk + dt * ak : v_m1[3 * i + k] + 2.0 * dt * ak;
                r[3 * i + k] = r[3 * i + k] + dt * vk + 0.5 * dt * dt * ak;
                v_m1[3 * i + k] = vk;
                v[3 * i + k] = v_new;
            }
        } else {
            for (int k = 0; k < 3; ++k) v_m1[3 * i + k] = v[3 * i + k];
        }
        rho_m1[i] = rho[i];
        rho[i] = rho_new;
    }
}

/* One full step n (0-based): rates at the pre-update state, then Verlet.
 * acc/drho receive the rates used. */
int orc_step(const orc_params *P, long n, double *r, double *v, double *rho,
             double *v_m1, double *rho_m1, const unsigned char *type,
             double dt, long step_index, int verlet_ns, int mode, double *acc, double *drho)
{
    int rc = orc_rates(P, n, r, v, rho, type, NULL, mode, acc, drho);
    if (rc) return rc;
    int corrective = (verlet_ns <= 0) ? (step_index == 0) : (step_index % verlet_ns == 0);
    orc_verlet(n, r, v, rho, v_m1, rho_m1, type, acc, drho, dt, corrective);
    return 0;
}
