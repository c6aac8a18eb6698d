/*
 * oracle/lv_oracle.c  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the per-timestep Langevin update of
 * Derkachov et al., "A numerical toy model of Langevin dynamics provides
 * real-time visualization of colloidal microdroplet evaporation"
 * (arxiv 2501.04456; /root/reference/PAPER.md).  It exists so that the CUDA
 * path (paper_2501_04456_b200/csrc) can be compared with something written
 * independently from the paper.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no
 * code, header, table or constant generator with the CUDA path.
 *
 * What follows the paper, and where:
 *   loop order (i)..(vi)                      PAPER.md:62-69 (sec. 2.2)
 *   LJ + Coulomb, truncated and NOT shifted
 *   interaction range per pair of NP radii
 *   radius update, radius-square law
 *   surface spring, equilibrium one NP radius
 *     inside the interface, per-type constant PAPER.md:58
 *   gravity, Stokes viscosity, centrifugal
 *   new velocity and position + random kick
 * The paper prints no formula for any of these; the formulas are the readings
 * listed in DESIGN.md ("Readings of the paper"), cited below as DESIGN R<n>.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): O(N^2) brute force vs the cell
 * list, Newton's third law, LJ dimer closed forms, Coulomb closed form,
 * energy conservation with drag/noise off, terminal velocity, equipartition,
 * Stokes-Einstein MSD closed form, wall statics, schedule closed forms,
 * Philox4x32-10 known answers, Gaussian moments.
 * "parity unpinned": the model as a whole against reality or against the
 * authors' program -- the paper prints no trajectory, energy or statistic in
 * text, so nothing can pin that.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -fPIC -shared (see
 * oracle/build.py).  -ffp-contract=off matters: the three "fp32 contract"
 * expressions below must be evaluated exactly as written.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define LVO_MAX_TYPES 8
#define LVO_PI 3.14159265358979323846

/* Everything that defines a simulation, in the paper's terms (PAPER.md:58:
 * "radius, mass, charge" per NP type, per-type spring constant, free
 * interaction matrix, evaporation rate, rotation, kick magnitude).
 * Pair tables are [a*LVO_MAX_TYPES + b]. */
typedef struct {
    int32_t  n_types;
    int32_t  wall_mode;   /* 0: one-sided spring (DESIGN R7); 1: paper's literal window */
    int32_t  sched_mode;  /* 0 const, 1 linear in n, 2 radius-square law (DESIGN R10) */
    int32_t  pad_;
    int64_t  sched_steps;
    uint64_t seed;
    double   dt;
    double   R0, R1;
    double   coulomb_k;   /* k_C in U = k_C q_a q_b / r (DESIGN R5) */
    double   g;           /* gravity along -z (DESIGN R13) */
    double   omega2[3];   /* centrifugal weights (DESIGN R14) */
    double   sigma[LVO_MAX_TYPES];   /* NP diameter, r_NP = sigma/2 */
    double   mass[LVO_MAX_TYPES];
    double   charge[LVO_MAX_TYPES];
    double   wall_k[LVO_MAX_TYPES];
    double   drag_a[LVO_MAX_TYPES];  /* per-step velocity retention a (DESIGN R11) */
    double   kick_b[LVO_MAX_TYPES];  /* per-component kick std b (DESIGN R15) */
    double   eps[LVO_MAX_TYPES * LVO_MAX_TYPES];
    double   sig[LVO_MAX_TYPES * LVO_MAX_TYPES];
    double   rcut[LVO_MAX_TYPES * LVO_MAX_TYPES];
} lvo_params;

/* ------------------------------------------------------------------ */
/* Parameter helpers                                                   */
/* ------------------------------------------------------------------ */

/* DESIGN R2/R3/R4: sigma_ab = r_a + r_b (PAPER.md:64 writes the range with
 * r_A + r_B), eps_ab = sqrt(eps_a eps_b), r_c,ab = cut_factor * sigma_ab
 * (range 4(r_A + r_B) = 4 sigma_ab, "can be changed"). */
void lvo_mix_lorentz_berthelot(lvo_params *p, const double *eps_a, double cut_factor)
{
    for (int a = 0; a < p->n_types; ++a)
        for (int b = 0; b < p->n_types; ++b) {
            int k = a * LVO_MAX_TYPES + b;
            p->sig[k]  = 0.5 * p->sigma[a] + 0.5 * p->sigma[b];
            p->eps[k]  = sqrt(eps_a[a] * eps_a[b]);
            p->rcut[k] = cut_factor * p->sig[k];
        }
}

/* DESIGN R11/R15: explicit Stokes drag a = 1 - gamma dt;
 * kick b = sqrt((kT/m)(1 - a^2)) makes <v^2> = kT/m stationary (PAPER.md:69:
 * the kick magnitude "imposes [temperature] externally"). */
void lvo_langevin_coeffs(double gamma, double kT, double mass, double dt,
                         double *a, double *b)
{
    *a = 1.0 - gamma * dt;
    *b = sqrt((kT / mass) * (1.0 - (*a) * (*a)));
}

/* Step (iii); DESIGN R10, R27: R is a function of the integer
 * step index. */
double lvo_radius(const lvo_params *p, int64_t n)
{
    if (p->sched_mode == 0 || p->sched_steps <= 0) return p->R0;
    int64_t m = n < 0 ? 0 : (n > p->sched_steps ? p->sched_steps : n);
    double f = (double)m / (double)p->sched_steps;
    if (m == p->sched_steps) return p->R1;
    if (p->sched_mode == 1) return p->R0 + (p->R1 - p->R0) * f;
    return sqrt(p->R0 * p->R0 + (p->R1 * p->R1 - p->R0 * p->R0) * f);
}

/* ------------------------------------------------------------------ */
/* Pair force, step (ii)                                               */
/* ------------------------------------------------------------------ */

/* fp32 contract expression #2 (DESIGN "fp32 contracts"): the in-range
 * predicate is defined on the fp32 state by this exact sequence, so that
 * neighbour counts are bit-exact between the two sides.  Strict '<'
 * (truncated, zero at and beyond the range). */
static int in_range_f32(const float *xi, const float *xj, float rc2)
{
    float dx = xi[0] - xj[0];
    float dy = xi[1] - xj[1];
    float dz = xi[2] - xj[2];
    float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    return r2 < rc2;
}

/* One ordered pair i<-j.  DESIGN R1: U = 4 eps [(s/r)^12 - (s/r)^6];
 * DESIGN R5: U_C = k_C q_a q_b / r; no shift of force or energy.
 *   F_ij = [ 24 eps (2 s6^2 - s6)/r^2 + k_C q_a q_b / r^3 ] (x_i - x_j)
 * acc[0..2] += F, acc[3] += sum of the three term magnitudes, acc[4] += U. */
static void pair_term(const lvo_params *p, int a, int b,
                      const double *xi, const double *xj, double *acc)
{
    int k = a * LVO_MAX_TYPES + b;
    double dx = xi[0] - xj[0], dy = xi[1] - xj[1], dz = xi[2] - xj[2];
    double r2 = dx * dx + dy * dy + dz * dz;
    double r = sqrt(r2);
    double s2 = p->sig[k] * p->sig[k] / r2;
    double s6 = s2 * s2 * s2;
    double rep = 48.0 * p->eps[k] * s6 * s6 / r2;
    double att = 24.0 * p->eps[k] * s6 / r2;
    double qq = p->coulomb_k * p->charge[a] * p->charge[b];
    double cou = qq / (r2 * r);
    double f = rep - att + cou;
    acc[0] += f * dx;
    acc[1] += f * dy;
    acc[2] += f * dz;
    acc[3] += (fabs(rep) + fabs(att) + fabs(cou)) * r;
    acc[4] += 4.0 * p->eps[k] * (s6 * s6 - s6) + qq / r;
}

static void to_f32(int n, const double *x, float *xf)
{
    for (int i = 0; i < 3 * n; ++i) xf[i] = (float)x[i];
}

/* The definition: the plain O(N^2) sum over all j != i inside the pair's
 * range.  F[N][3], S[N] (sum of term magnitudes, the parity
 * denominator), cnt[N] (in-range neighbours), returns total pair energy
 * (each unordered pair once).  Any output pointer may be NULL. */
double lvo_pair_forces_brute(const lvo_params *p, int n, const double *x,
                             const int32_t *type, double *F, double *S, int32_t *cnt)
{
    float *xf = (float *)malloc(sizeof(float) * 3 * (size_t)n);
    to_f32(n, x, xf);
    double U = 0.0;
#pragma omp parallel for schedule(dynamic, 32) reduction(+ : U)
    for (int i = 0; i < n; ++i) {
        double acc[5] = {0, 0, 0, 0, 0};
        int c = 0;
        for (int j = 0; j < n; ++j) {
            if (j == i) continue;
            double rc = p->rcut[type[i] * LVO_MAX_TYPES + type[j]];
            float rc2 = (float)(rc * rc);
            if (!in_range_f32(xf + 3 * i, xf + 3 * j, rc2)) continue;
            pair_term(p, type[i], type[j], x + 3 * i, x + 3 * j, acc);
            ++c;
        }
        if (F) { F[3 * i] = acc[0]; F[3 * i + 1] = acc[1]; F[3 * i + 2] = acc[2]; }
        if (S) S[i] = acc[3];
        if (cnt) cnt[i] = c;
        U += 0.5 * acc[4];
    }
    free(xf);
    return U;
}

/* Step (i): cells exist only "to identify which [NPs] are close
 * to each other and can interact" -- a faster route to the same sum.  The
 * oracle's own structure is a head/next linked list on one grid of edge
 * max r_c over the bounding box of the positions, binned in fp64.  Checked
 * against lvo_pair_forces_brute in tests/test_oracle_forces.py. */
double lvo_pair_forces_cells(const lvo_params *p, int n, const double *x,
                             const int32_t *type, double *F, double *S, int32_t *cnt)
{
    if (n <= 0) return 0.0;
    double rcmax = 0.0;
    for (int a = 0; a < p->n_types; ++a)
        for (int b = 0; b < p->n_types; ++b)
            if (p->rcut[a * LVO_MAX_TYPES + b] > rcmax) rcmax = p->rcut[a * LVO_MAX_TYPES + b];
    double lo[3], hi[3];
    for (int d = 0; d < 3; ++d) { lo[d] = x[d]; hi[d] = x[d]; }
    for (int i = 0; i < n; ++i)
        for (int d = 0; d < 3; ++d) {
            if (x[3 * i + d] < lo[d]) lo[d] = x[3 * i + d];
            if (x[3 * i + d] > hi[d]) hi[d] = x[3 * i + d];
        }
    double h = rcmax * 1.001;   /* margin: the fp32 predicate may pass r slightly above r_c */
    int G[3];
    for (int d = 0; d < 3; ++d) {
        double g = floor((hi[d] - lo[d]) / h) + 1.0;
        double cap = ceil(cbrt(4.0 * (double)n)) + 4.0;   /* about 4 cells per NP at most; */
        if (g > cap) g = cap;                             /* cells only get coarser       */
        G[d] = (int)g;
    }
    double hh[3];
    for (int d = 0; d < 3; ++d) {
        hh[d] = (hi[d] - lo[d]) / G[d];
        if (hh[d] < h) hh[d] = h;
    }
    size_t ncell = (size_t)G[0] * G[1] * G[2];
    int *head = (int *)malloc(sizeof(int) * ncell);
    int *next = (int *)malloc(sizeof(int) * (size_t)n);
    int *cell = (int *)malloc(sizeof(int) * 3 * (size_t)n);
    for (size_t c = 0; c < ncell; ++c) head[c] = -1;
    for (int i = 0; i < n; ++i) {
        int c[3];
        for (int d = 0; d < 3; ++d) {
            double t = floor((x[3 * i + d] - lo[d]) / hh[d]);
            c[d] = (t >= 0.0 && t < 1e9) ? (int)t : 0;   /* NaN, inf -> cell 0 */
            if (c[d] > G[d] - 1) c[d] = G[d] - 1;
            cell[3 * i + d] = c[d];
        }
        size_t k = ((size_t)c[2] * G[1] + c[1]) * G[0] + c[0];
        next[i] = head[k];
        head[k] = i;
    }
    float *xf = (float *)malloc(sizeof(float) * 3 * (size_t)n);
    to_f32(n, x, xf);
    double U = 0.0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : U)
    for (int i = 0; i < n; ++i) {
        double acc[5] = {0, 0, 0, 0, 0};
        int c = 0;
        for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
            int cx = cell[3 * i] + dx, cy = cell[3 * i + 1] + dy, cz = cell[3 * i + 2] + dz;
            if (cx < 0 || cy < 0 || cz < 0 || cx >= G[0] || cy >= G[1] || cz >= G[2]) continue;
            size_t k = ((size_t)cz * G[1] + cy) * G[0] + cx;
            for (int j = head[k]; j >= 0; j = next[j]) {
                if (j == i) continue;
                double rc = p->rcut[type[i] * LVO_MAX_TYPES + type[j]];
                float rc2 = (float)(rc * rc);
                if (!in_range_f32(xf + 3 * i, xf + 3 * j, rc2)) continue;
                pair_term(p, type[i], type[j], x + 3 * i, x + 3 * j, acc);
                ++c;
            }
        }
        if (F) { F[3 * i] = acc[0]; F[3 * i + 1] = acc[1]; F[3 * i + 2] = acc[2]; }
        if (S) S[i] = acc[3];
        if (cnt) cnt[i] = c;
        U += 0.5 * acc[4];
    }
    free(xf); free(cell); free(next); free(head);
    return U;
}

/* ------------------------------------------------------------------ */
/* Surface and external forces, steps (iv) and (v)                      */
/* ------------------------------------------------------------------ */

/* Step (iv): spring with its equilibrium point one
 * NP radius inside the interface.  DESIGN R7: pen = |x| - (R - r_a);
 * F = -k_a pen x/|x| for pen > 0 (wall_mode 1: only while pen < 2 r_a, the
 * paper's (-r_NP, r_NP) window around the surface).
 * Step (v): gravity -m g z^ (DESIGN R13) and
 * centrifugal m (O2x x, O2y y, O2z z) (DESIGN R14).  Drag enters through a_a
 * in the update.  F[N][3] is overwritten; S[N] receives |F_wall| + |F_g| +
 * |F_c|; returns the potential energy of these terms. */
double lvo_external_forces(const lvo_params *p, double R, int n, const double *x,
                           const int32_t *type, double *F, double *S)
{
    double U = 0.0;
    for (int i = 0; i < n; ++i) {
        int a = type[i];
        const double *xi = x + 3 * i;
        double m = p->mass[a];
        double f[3] = {0, 0, 0};
        double r = sqrt(xi[0] * xi[0] + xi[1] * xi[1] + xi[2] * xi[2]);
        double ra = 0.5 * p->sigma[a];
        double pen = r - (R - ra);
        double fw = 0.0;
        if (pen > 0.0 && r > 0.0 && (p->wall_mode == 0 || pen < 2.0 * ra)) {
            fw = p->wall_k[a] * pen;
            for (int d = 0; d < 3; ++d) f[d] -= fw * xi[d] / r;
            U += 0.5 * p->wall_k[a] * pen * pen;
        }
        double fg = m * p->g;
        f[2] -= fg;
        U += m * p->g * xi[2];
        double fc[3];
        for (int d = 0; d < 3; ++d) {
            fc[d] = m * p->omega2[d] * xi[d];
            f[d] += fc[d];
            U -= 0.5 * m * p->omega2[d] * xi[d] * xi[d];
        }
        if (F) { F[3 * i] = f[0]; F[3 * i + 1] = f[1]; F[3 * i + 2] = f[2]; }
        if (S) S[i] = fabs(fw) + fabs(fg) + sqrt(fc[0] * fc[0] + fc[1] * fc[1] + fc[2] * fc[2]);
    }
    return U;
}

/* ------------------------------------------------------------------ */
/* Brownian kick, step (vi)                                             */
/* ------------------------------------------------------------------ */

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): counter-based, so the
 * GPU side can draw the identical numbers from (id, step) alone.  Pinned by
 * the published known-answer vectors in tests/golden/philox4x32_10_kat.txt. */
void lvo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* DESIGN R15: "a randomly directed vector, whose magnitude can be controlled"
 * = three iid unit Gaussians (isotropic direction), scaled
 * by b_a in the update.  key = (seed_lo, seed_hi), counter = (id, n_lo, n_hi,
 * 0): keyed on the particle's id and the step index, never on a slot.
 * u = ((w >> 9) + 0.5) 2^-23 lies in (0,1) and is exact in fp32 and fp64. */
void lvo_gauss3(uint64_t seed, uint32_t id, int64_t step, double xi[3])
{
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t ctr[4] = {id, (uint32_t)(uint64_t)step, (uint32_t)((uint64_t)step >> 32), 0u};
    uint32_t w[4];
    lvo_philox4x32_10(ctr, key, w);
    double u[4];
    for (int k = 0; k < 4; ++k) u[k] = ((double)(w[k] >> 9) + 0.5) * (1.0 / 8388608.0);
    double r01 = sqrt(-2.0 * log(u[0]));
    double r23 = sqrt(-2.0 * log(u[2]));
    xi[0] = r01 * cos(2.0 * LVO_PI * u[1]);
    xi[1] = r01 * sin(2.0 * LVO_PI * u[1]);
    xi[2] = r23 * cos(2.0 * LVO_PI * u[3]);
}

void lvo_gauss3_batch(uint64_t seed, int n, const uint32_t *ids, int64_t step, double *xi)
{
    for (int i = 0; i < n; ++i) lvo_gauss3(seed, ids[i], step, xi + 3 * i);
}

/* ------------------------------------------------------------------ */
/* The step, PAPER.md:62-69 in the paper's order                        */
/* ------------------------------------------------------------------ */

/* Advances (x, v) in place from step index step0 by nsteps steps.
 * Particle id = row index.  use_cells selects the cell-list route to the
 * pair sum (same result).  Optional outputs of the LAST step taken:
 * Fpair[N][3], Fext[N][3].  Returns 0, or 1 if a non-finite value appeared. */
int lvo_step(const lvo_params *p, int n, double *x, double *v, const int32_t *type,
             int64_t step0, int nsteps, int use_cells, double *Fpair_out, double *Fext_out)
{
    double *Fp = (double *)malloc(sizeof(double) * 3 * (size_t)(n > 0 ? n : 1));
    double *Fe = (double *)malloc(sizeof(double) * 3 * (size_t)(n > 0 ? n : 1));
    int bad = 0;
    for (int s = 0; s < nsteps; ++s) {
        int64_t nidx = step0 + s;
        /* (i)+(ii): cells and pair forces from x_n */
        if (use_cells) lvo_pair_forces_cells(p, n, x, type, Fp, NULL, NULL);
        else           lvo_pair_forces_brute(p, n, x, type, Fp, NULL, NULL);
        /* (iii): new radius -- before the surface force, so the wall of step n
         * stands at R(n+1) (DESIGN R9) */
        double Rn = lvo_radius(p, nidx + 1);
        /* (iv)+(v) */
        lvo_external_forces(p, Rn, n, x, type, Fe, NULL);
        /* (vi): v <- a v + (dt/m) F + b xi ; x <- x + dt v  (DESIGN R16:
         * semi-implicit Euler, the position uses the new velocity) */
        for (int i = 0; i < n; ++i) {
            int a = type[i];
            double xi[3];
            lvo_gauss3(p->seed, (uint32_t)i, nidx, xi);
            for (int d = 0; d < 3; ++d) {
                double F = Fp[3 * i + d] + Fe[3 * i + d];
                double vn = p->drag_a[a] * v[3 * i + d] + (p->dt / p->mass[a]) * F
                          + p->kick_b[a] * xi[d];
                v[3 * i + d] = vn;
                x[3 * i + d] += p->dt * vn;
                if (!isfinite(vn) || !isfinite(x[3 * i + d])) bad = 1;
            }
        }
    }
    if (Fpair_out && nsteps > 0) memcpy(Fpair_out, Fp, sizeof(double) * 3 * (size_t)n);
    if (Fext_out && nsteps > 0) memcpy(Fext_out, Fe, sizeof(double) * 3 * (size_t)n);
    free(Fp); free(Fe);
    return bad;
}

/* E = sum 1/2 m v^2 + U_pair + U_wall + U_g + U_c at radius R.
 * out[0] = kinetic, out[1] = pair, out[2] = wall + gravity + centrifugal. */
void lvo_energy(const lvo_params *p, double R, int n, const double *x, const double *v,
                const int32_t *type, double out[3])
{
    double ke = 0.0;
    for (int i = 0; i < n; ++i) {
        double m = p->mass[type[i]];
        ke += 0.5 * m * (v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2]);
    }
    out[0] = ke;
    out[1] = lvo_pair_forces_brute(p, n, x, type, NULL, NULL, NULL);
    out[2] = lvo_external_forces(p, R, n, x, type, NULL, NULL);
}

/* ------------------------------------------------------------------ */
/* fp32 contracts for the cell structures (steps A2-A4)                 */
/* ------------------------------------------------------------------ */

/* DESIGN "Grid rule".  One uniform grid per NP type b over the cube
 * [-L_b, L_b]^3, particles binned on the grid of their own type, key space
 * laid out type-major.  All derived in fp64 and rounded once to fp32. */
typedef struct {
    int32_t  n_types;
    int32_t  G[LVO_MAX_TYPES];          /* cells per axis of grid b */
    uint32_t base[LVO_MAX_TYPES + 1];   /* first key of grid b; base[T] = total cells */
    float    lo[LVO_MAX_TYPES];         /* lower corner (all three axes) */
    float    inv_h[LVO_MAX_TYPES];
    double   h[LVO_MAX_TYPES];
    int32_t  w[LVO_MAX_TYPES * LVO_MAX_TYPES]; /* stencil half-width, target a in grid b */
} lvo_grid;

/* h_b = r_c,bb (1 + 2^-9) / k_b, k_b = cells per cut-off (>= 1);
 * G_b = ceil((2 R_max + 2 sigma_max) / h_b);  lo_b = -G_b h_b / 2;
 * w_ab = ceil(r_c,ab (1 + 2^-10) / h_b). */
void lvo_grid_spec(const lvo_params *p, const int32_t *cells_per_cut, lvo_grid *g)
{
    double Rmax = p->sched_mode == 0 ? p->R0 : (p->R0 > p->R1 ? p->R0 : p->R1);
    double smax = 0.0;
    for (int a = 0; a < p->n_types; ++a) if (p->sigma[a] > smax) smax = p->sigma[a];
    memset(g, 0, sizeof(*g));
    g->n_types = p->n_types;
    uint32_t base = 0;
    for (int b = 0; b < p->n_types; ++b) {
        int k = cells_per_cut ? cells_per_cut[b] : 1;
        double h = p->rcut[b * LVO_MAX_TYPES + b] * (1.0 + 1.0 / 512.0) / (double)k;
        int G = (int)ceil((2.0 * Rmax + 2.0 * smax) / h);
        g->h[b] = h;
        g->G[b] = G;
        g->lo[b] = (float)(-0.5 * (double)G * h);
        g->inv_h[b] = (float)(1.0 / h);
        g->base[b] = base;
        base += (uint32_t)G * (uint32_t)G * (uint32_t)G;
    }
    g->base[p->n_types] = base;
    for (int a = 0; a < p->n_types; ++a)
        for (int b = 0; b < p->n_types; ++b)
            g->w[a * LVO_MAX_TYPES + b] =
                (int)ceil(p->rcut[a * LVO_MAX_TYPES + b] * (1.0 + 1.0 / 1024.0) / g->h[b]);
}

/* fp32 contract expression #1: t = fl32(fl32(x - lo) * inv_h);
 * c = clamp(floor(t), 0, G-1), NaN -> 0.  Clamp, not wrap: a droplet is not
 * periodic. */
static int cell_coord_f32(float x, float lo, float inv_h, int G)
{
    float t = (x - lo) * inv_h;
    float f = floorf(t);
    if (!(f >= 0.0f)) return 0;
    if (f > (float)(G - 1)) return G - 1;
    return (int)f;
}

/* key = base[type] + (c_z G + c_y) G + c_x on the grid of the NP's own type. */
void lvo_cell_keys(const lvo_grid *g, int n, const float *x, const int32_t *type, uint32_t *key)
{
    for (int i = 0; i < n; ++i) {
        int b = type[i];
        int G = g->G[b];
        int cx = cell_coord_f32(x[3 * i], g->lo[b], g->inv_h[b], G);
        int cy = cell_coord_f32(x[3 * i + 1], g->lo[b], g->inv_h[b], G);
        int cz = cell_coord_f32(x[3 * i + 2], g->lo[b], g->inv_h[b], G);
        key[i] = g->base[b] + (uint32_t)((cz * G + cy) * G + cx);
    }
}

/* contract #3: STABLE sort by key; ties keep the current order. */
typedef struct { uint32_t key, idx; } kv_t;
static int kv_cmp(const void *a, const void *b)
{
    const kv_t *p = (const kv_t *)a, *q = (const kv_t *)b;
    if (p->key != q->key) return p->key < q->key ? -1 : 1;
    return p->idx < q->idx ? -1 : (p->idx > q->idx ? 1 : 0);
}
void lvo_stable_sort_perm(int n, const uint32_t *key, uint32_t *key_sorted, uint32_t *perm)
{
    kv_t *kv = (kv_t *)malloc(sizeof(kv_t) * (size_t)(n > 0 ? n : 1));
    for (int i = 0; i < n; ++i) { kv[i].key = key[i]; kv[i].idx = (uint32_t)i; }
    qsort(kv, (size_t)n, sizeof(kv_t), kv_cmp);
    for (int i = 0; i < n; ++i) { key_sorted[i] = kv[i].key; perm[i] = kv[i].idx; }
    free(kv);
}

/* off[c] = number of sorted keys < c, c = 0..n_cells: cell c holds the sorted
 * slots [off[c], off[c+1]). */
void lvo_cell_offsets(int n, const uint32_t *key_sorted, uint32_t n_cells, uint32_t *off)
{
    uint32_t k = 0;
    for (uint32_t c = 0; c <= n_cells; ++c) {
        while (k < (uint32_t)n && key_sorted[k] < c) ++k;
        off[c] = k;
    }
}


/* ------------------------------------------------------------------ */
/* Observables as integer histograms.  The bin of a distance
 * is an integer decided by floating point, so -- as for the cell hash -- it is DEFINED
 * on the fp32 state by a fixed fp32 expression that both sides evaluate literally
 * (fp32 contract #4):
 *     r2 as in contract #2;  r = sqrtf(r2) (correctly rounded);
 *     bin = (int) fl32(r * inv_dr),  inv_dr = fl32(1 / dr);  counted iff bin < n_bins.
 * The histograms below are the plain definitions: every ordered pair (Eq. 6: each NP
 * in turn is the "trial particle"), every NP (Eq. 8).
 * They are pinned against oracle/observables.py (fp64, np.histogram), itself pinned
 * against closed forms. */
void lvo_rdf_hist(int n, const float *x, float inv_dr, int n_bins, uint64_t *hist)
{
    for (int b = 0; b < n_bins; ++b) hist[b] = 0;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) {
            if (j == i) continue;
            float dx = x[3 * i] - x[3 * j];
            float dy = x[3 * i + 1] - x[3 * j + 1];
            float dz = x[3 * i + 2] - x[3 * j + 2];
            float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            float t = sqrtf(r2) * inv_dr;
            if (t < (float)n_bins) hist[(int)t] += 1;
        }
}

/* Eq. 8 numerator psi(r_sun) per shell around the droplet centre, the sums of Eq. 3-4
 * (sum x, sum |x|^2, fp64 from the fp32 state) and N_surf: NPs whose surface is
 * within one NP radius of the interface, |x| > R - 2 r_a, decided in fp64. */
void lvo_radial_hist(int n, const float *x, const int32_t *type, const double *radius_a,
                     double R, float inv_dr, int n_bins, uint64_t *hist, double sums[4],
                     int64_t *n_surf)
{
    for (int b = 0; b < n_bins; ++b) hist[b] = 0;
    sums[0] = sums[1] = sums[2] = sums[3] = 0.0;
    *n_surf = 0;
    for (int i = 0; i < n; ++i) {
        float fx = x[3 * i], fy = x[3 * i + 1], fz = x[3 * i + 2];
        float t = sqrtf(fmaf(fz, fz, fmaf(fy, fy, fx * fx))) * inv_dr;
        if (t < (float)n_bins) hist[(int)t] += 1;
        double dx = fx, dy = fy, dz = fz;
        double r2 = dx * dx + dy * dy + dz * dz;
        sums[0] += dx; sums[1] += dy; sums[2] += dz; sums[3] += r2;
        if (sqrt(r2) > R - 2.0 * radius_a[type[i]]) *n_surf += 1;
    }
}

/* Aggregates (reading R23): connected components of the bond graph r2 < rb2_ab, r2 by
 * contract #2 on the fp32 state, rb2 a T x T fp32 table (row stride LVO_MAX_TYPES) of
 * squared bond lengths.  Plain O(N^2) union by relabelling: label[i] = smallest index of
 * i's component. */
void lvo_cluster_labels(int n, const float *x, const int32_t *type, const float *rb2,
                        int32_t *label)
{
    for (int i = 0; i < n; ++i) label[i] = i;
    int changed = 1;
    while (changed) {               /* propagate the minimum label along bonds until stable */
        changed = 0;
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j) {
                if (j == i || label[j] >= label[i]) continue;
                if (in_range_f32(x + 3 * i, x + 3 * j, rb2[type[i] * LVO_MAX_TYPES + type[j]])) {
                    label[i] = label[j];
                    changed = 1;
                }
            }
    }
}

/* ------------------------------------------------------------------ */
/* Headless perspective view (Fig. 2 right panel).
 * Plain restatement of the splat: per NP, per pixel of its bounding box, single fp32
 * operations in the order include/lv.h states (this file is built with
 * -ffp-contract=off); the nearest fragment wins, ties by the smaller pixel value.
 * rot: 9 floats row-major; palette / radius: per type. */
static uint32_t shade_px(uint32_t base, float s)
{
    uint32_t out = 0xff000000u;
    for (int c = 0; c < 3; ++c) {
        float ch = (float)((base >> (8 * c)) & 0xffu);
        uint32_t q = (uint32_t)(ch * s + 0.5f);
        out |= (q > 255u ? 255u : q) << (8 * c);
    }
    return out;
}

void lvo_render(int n, const float *x, const int32_t *type, const float *radius_a,
                const float *rot, float eye, float focal, int width, int height,
                const uint32_t *palette, uint32_t background, uint32_t droplet, float R,
                uint32_t *rgba)
{
    size_t n_px = (size_t)width * height;
    uint64_t *zb = (uint64_t *)malloc(8 * n_px);
    for (size_t p = 0; p < n_px; ++p) zb[p] = ~(uint64_t)0;
    float cx = (float)(0.5 * width), cy = (float)(0.5 * height);
    for (int i = 0; i < n; ++i) {
        float px_ = x[3 * i], py_ = x[3 * i + 1], pz_ = x[3 * i + 2];
        float r = radius_a[type[i]];
        float xc = (rot[0] * px_ + rot[1] * py_) + rot[2] * pz_;
        float yc = (rot[3] * px_ + rot[4] * py_) + rot[5] * pz_;
        float zr = (rot[6] * px_ + rot[7] * py_) + rot[8] * pz_;
        float zc = eye - zr;
        if (!(zc > 2.0f * r)) continue;
        float inv = focal / zc;
        float u = cx + xc * inv;
        float v = cy - yc * inv;
        float rho = r * inv;
        float rho2 = rho * rho;
        if (!(rho2 > 0.0f) || !(fabsf(u) < 1e7f) || !(fabsf(v) < 1e7f) || !(rho < 1e4f)) continue;
        int x0 = (int)floorf(u - rho), x1 = (int)floorf(u + rho);
        int y0 = (int)floorf(v - rho), y1 = (int)floorf(v + rho);
        if (x0 < 0) x0 = 0;
        if (y0 < 0) y0 = 0;
        if (x1 > width - 1) x1 = width - 1;
        if (y1 > height - 1) y1 = height - 1;
        for (int py = y0; py <= y1; ++py) {
            float dy = ((float)py + 0.5f) - v;
            float dy2 = dy * dy;
            for (int px = x0; px <= x1; ++px) {
                float dx = ((float)px + 0.5f) - u;
                float d2 = dx * dx + dy2;
                if (d2 <= rho2) {
                    float nz = sqrtf((rho2 - d2) / rho2);
                    float zf = zc - r * nz;
                    uint32_t c = shade_px(palette[type[i]], 0.25f + 0.75f * nz);
                    uint32_t zbits;
                    memcpy(&zbits, &zf, 4);
                    uint64_t key = ((uint64_t)zbits << 32) | c;
                    size_t p = (size_t)py * width + px;
                    if (key < zb[p]) zb[p] = key;
                }
            }
        }
    }
    float rr = R * (focal / eye);
    for (int py = 0; py < height; ++py)
        for (int px = 0; px < width; ++px) {
            size_t p = (size_t)py * width + px;
            if (zb[p] != ~(uint64_t)0) { rgba[p] = (uint32_t)zb[p]; continue; }
            float dx = ((float)px + 0.5f) - cx, dy = ((float)py + 0.5f) - cy;
            float d2 = dx * dx + dy * dy;
            rgba[p] = d2 <= rr * rr ? droplet : background;
        }
    free(zb);
}

/* The same view written as its DEFINITION, pixel by pixel: for EVERY pixel, EVERY NP is projected
 * and tested -- no bounding boxes, no per-NP pixel loops -- and the nearest fragment is kept.
 * O(pixels x NPs): small frames only.  lvo_render (the per-NP form the CUDA splat mirrors) must
 * give the same image bit for bit; a mistake in its bounding-box logic cannot hide here. */
void lvo_render_pixels(int n, const float *x, const int32_t *type, const float *radius_a,
                       const float *rot, float eye, float focal, int width, int height,
                       const uint32_t *palette, uint32_t background, uint32_t droplet, float R,
                       uint32_t *rgba)
{
    float cx = (float)(0.5 * width), cy = (float)(0.5 * height);
    float rr = R * (focal / eye);
#pragma omp parallel for schedule(static)
    for (int py = 0; py < height; ++py)
        for (int px = 0; px < width; ++px) {
            uint64_t best = ~(uint64_t)0;
            for (int i = 0; i < n; ++i) {
                float px_ = x[3 * i], py_ = x[3 * i + 1], pz_ = x[3 * i + 2];
                float r = radius_a[type[i]];
                float xc = (rot[0] * px_ + rot[1] * py_) + rot[2] * pz_;
                float yc = (rot[3] * px_ + rot[4] * py_) + rot[5] * pz_;
                float zr = (rot[6] * px_ + rot[7] * py_) + rot[8] * pz_;
                float zc = eye - zr;
                if (!(zc > 2.0f * r)) continue;
                float inv = focal / zc;
                float u = cx + xc * inv;
                float v = cy - yc * inv;
                float rho = r * inv;
                float rho2 = rho * rho;
                if (!(rho2 > 0.0f) || !(fabsf(u) < 1e7f) || !(fabsf(v) < 1e7f) || !(rho < 1e4f)) continue;
                float dx = ((float)px + 0.5f) - u, dy = ((float)py + 0.5f) - v;
                float d2 = dx * dx + dy * dy;
                if (!(d2 <= rho2)) continue;
                float nz = sqrtf((rho2 - d2) / rho2);
                float zf = zc - r * nz;
                uint32_t c = shade_px(palette[type[i]], 0.25f + 0.75f * nz);
                uint32_t zbits;
                memcpy(&zbits, &zf, 4);
                uint64_t key = ((uint64_t)zbits << 32) | c;
                if (key < best) best = key;
            }
            size_t p = (size_t)py * width + px;
            if (best != ~(uint64_t)0) { rgba[p] = (uint32_t)best; continue; }
            float dx = ((float)px + 0.5f) - cx, dy = ((float)py + 0.5f) - cy;
            rgba[p] = dx * dx + dy * dy <= rr * rr ? droplet : background;
        }
}

/* Surface map, the left panel of Fig. 2 ("projection of the microdroplet
 * surface onto a plane", NP intersections with the surface as circles "elongated due to the
 * projection"); the projection is this build's reading (equirectangular, pole = z), its
 * definition is in include/lv.h.  Written as the definition: for EVERY pixel, the surface
 * point it looks at, then EVERY NP tested against it -- no windows, no culling.  The
 * direction factors are fp64 libm values rounded once to fp32; the coverage test is single
 * fp32 operations in the stated order (-ffp-contract=off). */
void lvo_render_surface(int n, const float *x, const int32_t *type, const float *radius_a,
                        float R, int width, int height, const uint32_t *palette,
                        uint32_t droplet, uint32_t *rgba)
{
    const double pi = 3.14159265358979323846;
#pragma omp parallel for schedule(static)
    for (int py = 0; py < height; ++py) {
        double phi = 0.5 * pi - pi * (((double)py + 0.5) / (double)height);
        float cl = (float)cos(phi), sl = (float)sin(phi);
        for (int px = 0; px < width; ++px) {
            double lam = -pi + (2.0 * pi) * (((double)px + 0.5) / (double)width);
            float co = (float)cos(lam), so = (float)sin(lam);
            float sx = R * (cl * co), sy = R * (cl * so), sz = R * sl;
            uint64_t best = ~(uint64_t)0;
            for (int i = 0; i < n; ++i) {
                float r = radius_a[type[i]];
                float dx = sx - x[3 * i], dy = sy - x[3 * i + 1], dz = sz - x[3 * i + 2];
                float d2 = (dx * dx + dy * dy) + dz * dz;
                if (d2 < r * r) {
                    uint32_t bits;
                    memcpy(&bits, &d2, 4);
                    uint64_t key = ((uint64_t)bits << 32) | (palette[type[i]] | 0xff000000u);
                    if (key < best) best = key;
                }
            }
            rgba[(size_t)py * width + px] = best == ~(uint64_t)0 ? droplet : (uint32_t)best;
        }
    }
}

int lvo_sizeof_params(void) { return (int)sizeof(lvo_params); }
int lvo_sizeof_grid(void) { return (int)sizeof(lvo_grid); }
int lvo_max_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
