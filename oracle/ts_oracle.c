/*
 * ts_oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 CPU oracle for the batched
 * pair-potential MD / FIRE hot path.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this file.  It shares no code, header, table or constant generator with the CUDA path
 * under paper_2508_06628_b200/csrc/ and neither includes the other.
 *
 * What the paper fixes: PAPER.md:29 (section 1, Abstract) names the potentials ("Lennard-Jones,
 * Morse, soft-sphere"), "molecular dynamics integrators" and "structural relaxation optimizers";
 * PAPER.md:56 (section 2) fixes the outputs "energies, forces, and stress"
 * (section 3) fixes the ragged batch (atom-wise attributes concatenated, system-wise stacked);
 * PAPER.md:92 (section 3) the per-system convergence check; PAPER.md:102 (section 4) Langevin MD.
 * The paper prints no formula for any of them; the formulas are the textbook definitions listed
 * as O1..O6 in SURVEY.md section 8(c) and the readings R1..R34 restated in DESIGN.md.
 *
 * Everything is the definition written out: O(N_s^2) search over all periodic images at every
 * force evaluation, no neighbour list, no skin, no cell list, no blocking, fixed loop order
 * (i ascending, j ascending, S lexicographic), per-system sums compensated (Neumaier), threads
 * split systems and never a sum.  Build: gcc -O2 -ffp-contract=off -fno-fast-math (see build.py).
 *
 * Pins (tests/test_oracle_*.py): closed-form dimers, FCC shell sums, F = -dE/dx and
 * W = -dE/dstrain by finite differences, Newton's third law, supercell / re-basis invariance,
 * brute-force pair enumeration over a fixed image cube, Philox known-answer vectors, NVE
 * reversibility + 2nd-order convergence + drift bounds (cfg1, cfg3), BAOAB limits and the Boltzmann
 * bond fluctuation of a Morse dimer, FIRE on a harmonic dimer, the FIRE velocity mixing on a
 * non-collinear cluster with the pre-update alpha (R21) and the P == 0 boundary, and Eabs against a
 * dimer and an independent lattice sum with V of both signs (tests/test_oracle_pins_r2.py).
 * No function of this file is "parity unpinned".
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_OK 0
#define ORC_ERR_ARG 1
#define ORC_ERR_CAP 2

enum { ORC_LJ = 0, ORC_MORSE = 1, ORC_SOFT = 2 };

typedef struct {
    int64_t n_atoms;
    int32_t n_systems;
    const int64_t *sys_off; /* [S+1] first atom of each system                              */
    double *pos;            /* [N,3] stored (never wrapped, R5) positions                   */
    double *vel;            /* [N,3]                                                        */
    double *force;          /* [N,3]                                                        */
    const double *mass;     /* [N]                                                          */
    const int32_t *type;    /* [N]                                                          */
    const double *cell;     /* [S,3,3] rows are lattice vectors (R4): x = f . h             */
    int32_t kind, n_types, shift_energy;
    const double *p0, *p1, *p2, *rc; /* [n_types*n_types] tables (O2)                       */
    double mass_conv, kB;   /* O3 units (R1)                                                */
} orc_batch;

typedef struct {
    double dt_start, dt_max, f_inc, f_dec, alpha_start, f_alpha, f_max;
    int32_t n_min, max_steps;
} orc_fire_params;

/* ---------------------------------------------------------------- compensated summation (O8) */
typedef struct { double s, c; } ksum;
static void kadd(ksum *k, double x)
{
    double t = k->s + x;
    if (fabs(k->s) >= fabs(x)) k->c += (k->s - t) + x;
    else                       k->c += (x - t) + k->s;
    k->s = t;
}
static double kval(const ksum *k) { return k->s + k->c; }

/* ---------------------------------------------------------------- O1: cell geometry           */
/* h[3*a+b] = component b of lattice vector a.  hinv = h^-1 so that f_k = sum_b x_b hinv[3b+k].
 * hperp_k = 1 / || column k of hinv ||  (distance between the lattice planes k).               */
int orc_cell_geometry(const double *h, double *hinv, double *hperp, double *vol)
{
    double c00 = h[4] * h[8] - h[5] * h[7];
    double c01 = h[5] * h[6] - h[3] * h[8];
    double c02 = h[3] * h[7] - h[4] * h[6];
    double det = h[0] * c00 + h[1] * c01 + h[2] * c02;
    if (!(fabs(det) > 0.0)) return ORC_ERR_ARG;
    hinv[0] = c00 / det;
    hinv[1] = (h[2] * h[7] - h[1] * h[8]) / det;
    hinv[2] = (h[1] * h[5] - h[2] * h[4]) / det;
    hinv[3] = c01 / det;
    hinv[4] = (h[0] * h[8] - h[2] * h[6]) / det;
    hinv[5] = (h[2] * h[3] - h[0] * h[5]) / det;
    hinv[6] = c02 / det;
    hinv[7] = (h[1] * h[6] - h[0] * h[7]) / det;
    hinv[8] = (h[0] * h[4] - h[1] * h[3]) / det;
    for (int k = 0; k < 3; ++k) {
        double n2 = hinv[k] * hinv[k] + hinv[3 + k] * hinv[3 + k] + hinv[6 + k] * hinv[6 + k];
        hperp[k] = 1.0 / sqrt(n2);
    }
    *vol = fabs(det);
    return ORC_OK;
}

/* ---------------------------------------------------------------- O1: pair enumeration         */
typedef void (*pair_cb)(void *ctx, int64_t i, int64_t j, const int32_t S[3], const double r[3],
                        double r2);

/* Directed pair set P(R) of one system: every ordered (i, j) including i == j, every integer
 * image S with |x_j - x_i + S.h|^2 < R^2 (strict), (i == j, S == 0) skipped.  The S range per
 * axis is the bound of O1; it is padded by a relative 1e-12 so rounding of the bound can never
 * drop an image the strict r^2 test would accept.                                              */
static int enumerate_pairs(const double *pos, int64_t n, const double *h, double R, pair_cb cb,
                           void *ctx)
{
    double hinv[9], hperp[3], vol;
    if (orc_cell_geometry(h, hinv, hperp, &vol) != ORC_OK) return ORC_ERR_ARG;
    double R2 = R * R;
    double w[3];
    for (int k = 0; k < 3; ++k) w[k] = (R / hperp[k]) * (1.0 + 1e-12) + 1e-12;
    for (int64_t i = 0; i < n; ++i) {
        for (int64_t j = 0; j < n; ++j) {
            double d[3], df[3];
            for (int b = 0; b < 3; ++b) d[b] = pos[3 * j + b] - pos[3 * i + b];
            for (int k = 0; k < 3; ++k)
                df[k] = d[0] * hinv[k] + d[1] * hinv[3 + k] + d[2] * hinv[6 + k];
            int32_t lo[3], hi[3];
            for (int k = 0; k < 3; ++k) {
                lo[k] = (int32_t)ceil(-df[k] - w[k]);
                hi[k] = (int32_t)floor(-df[k] + w[k]);
            }
            int32_t S[3];
            for (S[0] = lo[0]; S[0] <= hi[0]; ++S[0])
                for (S[1] = lo[1]; S[1] <= hi[1]; ++S[1])
                    for (S[2] = lo[2]; S[2] <= hi[2]; ++S[2]) {
                        if (i == j && S[0] == 0 && S[1] == 0 && S[2] == 0) continue;
                        double r[3];
                        for (int b = 0; b < 3; ++b)
                            r[b] = d[b] + ((double)S[0] * h[b] + (double)S[1] * h[3 + b] +
                                           (double)S[2] * h[6 + b]);
                        double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
                        if (r2 < R2) cb(ctx, i, j, S, r, r2);
                    }
        }
    }
    return ORC_OK;
}

typedef struct {
    int64_t cap, count;
    int32_t *oi, *oj, *oS;
    double *or2;
} list_ctx;

static void list_cb(void *vctx, int64_t i, int64_t j, const int32_t S[3], const double r[3],
                    double r2)
{
    list_ctx *c = (list_ctx *)vctx;
    (void)r;
    if (c->count < c->cap) {
        if (c->oi) c->oi[c->count] = (int32_t)i;
        if (c->oj) c->oj[c->count] = (int32_t)j;
        if (c->oS) { c->oS[3 * c->count] = S[0]; c->oS[3 * c->count + 1] = S[1]; c->oS[3 * c->count + 2] = S[2]; }
        if (c->or2) c->or2[c->count] = r2;
    }
    c->count++;
}

/* Export P(R) of one system.  Outputs may be NULL (count only).  Returns ORC_ERR_CAP when the
 * set does not fit cap (count still holds the true size).                                      */
int orc_pairs(const double *pos, int64_t n, const double *h, double R, int64_t cap, int32_t *oi,
              int32_t *oj, int32_t *oS, double *or2, int64_t *count)
{
    list_ctx c = { cap, 0, oi, oj, oS, or2 };
    int rc = enumerate_pairs(pos, n, h, R, list_cb, &c);
    if (rc != ORC_OK) return rc;
    *count = c.count;
    return (c.count > cap) ? ORC_ERR_CAP : ORC_OK;
}

/* ---------------------------------------------------------------- O2: potentials               */
static double ipow(double x, double a)
{
    double ia = floor(a);
    if (ia == a && a >= 0.0 && a <= 16.0) { /* small integer exponent: repeated multiplication */
        double r = 1.0;
        for (int k = 0; k < (int)ia; ++k) r *= x;
        return r;
    }
    return pow(x, a);
}

/* V(r) (unshifted) and V'(r) for one table entry.                                               */
static void pot_eval(int kind, double p0, double p1, double p2, double r, double *V, double *dV)
{
    if (kind == ORC_LJ) {            /* V = 4 eps [(s/r)^12 - (s/r)^6]                           */
        double sr = p1 / r, sr2 = sr * sr, sr6 = sr2 * sr2 * sr2, sr12 = sr6 * sr6;
        *V = 4.0 * p0 * (sr12 - sr6);
        *dV = -24.0 * p0 * (2.0 * sr12 - sr6) / r;
    } else if (kind == ORC_MORSE) {  /* V = D [(1 - e^{-a(r-r0)})^2 - 1]                         */
        double e = exp(-p1 * (r - p2));
        *V = p0 * ((1.0 - e) * (1.0 - e) - 1.0);
        *dV = 2.0 * p0 * p1 * (1.0 - e) * e;
    } else {                         /* V = (eps/alpha)(1 - r/sigma)^alpha, r < sigma            */
        double u = 1.0 - r / p1;
        if (u <= 0.0) { *V = 0.0; *dV = 0.0; return; }
        *V = (p0 / p2) * ipow(u, p2);
        *dV = -(p0 / p1) * ipow(u, p2 - 1.0);
    }
}

/* Public single-pair evaluation (used by the dimer pins): shifted energy and V'.               */
int orc_pair_potential(int kind, double p0, double p1, double p2, double rc, int shift_energy,
                       double r, double *V, double *dV)
{
    if (r >= rc) { *V = 0.0; *dV = 0.0; return ORC_OK; }
    pot_eval(kind, p0, p1, p2, r, V, dV);
    if (shift_energy) { double Vc, dVc; pot_eval(kind, p0, p1, p2, rc, &Vc, &dVc); *V -= Vc; }
    return ORC_OK;
}

typedef struct {
    const orc_batch *b;
    int64_t a0;          /* first atom of the system                                            */
    const double *vshift;/* [n_types^2] V(rc) or 0                                              */
    double *f;           /* force of atom i being accumulated (plain double, O8)                */
    int64_t cur_i;
    ksum E, Eabs, W[9];
} ef_ctx;

static void ef_cb(void *vctx, int64_t i, int64_t j, const int32_t S[3], const double r[3], double r2)
{
    ef_ctx *c = (ef_ctx *)vctx;
    const orc_batch *b = c->b;
    (void)S;
    int ti = b->type[c->a0 + i], tj = b->type[c->a0 + j];
    int t = ti * b->n_types + tj;
    double rc = b->rc[t];
    if (!(r2 < rc * rc)) return;           /* strict cutoff (R9): r >= rc contributes 0        */
    double rr = sqrt(r2), V, dV;
    pot_eval(b->kind, b->p0[t], b->p1[t], b->p2[t], rr, &V, &dV);
    V -= c->vshift[t];
    kadd(&c->E, 0.5 * V);
    kadd(&c->Eabs, 0.5 * fabs(V));
    double g = dV / rr;                    /* F_i = V'(r) r/|r|, r points i -> j               */
    double *f = b->force + 3 * (c->a0 + i);
    f[0] += g * r[0]; f[1] += g * r[1]; f[2] += g * r[2];
    for (int a = 0; a < 3; ++a)
        for (int d = 0; d < 3; ++d) kadd(&c->W[3 * a + d], -0.5 * g * r[a] * r[d]);
}

static double max_rc(const orc_batch *b)
{
    double m = 0.0;
    for (int t = 0; t < b->n_types * b->n_types; ++t) if (b->rc[t] > m) m = b->rc[t];
    return m;
}

/* E_s, F_i, W_s (O2) of one system; also Eabs = sum 1/2 |V| (scale for R31).                    */
static int system_energy_forces(const orc_batch *b, int s, const double *vshift, double *E,
                                double *W, double *Eabs)
{
    int64_t a0 = b->sys_off[s], n = b->sys_off[s + 1] - a0;
    ef_ctx c;
    memset(&c, 0, sizeof c);
    c.b = b; c.a0 = a0; c.vshift = vshift;
    for (int64_t i = 0; i < 3 * n; ++i) b->force[3 * a0 + i] = 0.0;
    int rc = enumerate_pairs(b->pos + 3 * a0, n, b->cell + 9 * s, max_rc(b), ef_cb, &c);
    if (rc != ORC_OK) return rc;
    if (E) *E = kval(&c.E);
    if (Eabs) *Eabs = kval(&c.Eabs);
    if (W) for (int k = 0; k < 9; ++k) W[k] = kval(&c.W[k]);
    return ORC_OK;
}

static double *make_vshift(const orc_batch *b)
{
    int nt = b->n_types * b->n_types;
    double *v = (double *)calloc((size_t)nt, sizeof(double));
    if (b->shift_energy)
        for (int t = 0; t < nt; ++t) {
            double dV;
            pot_eval(b->kind, b->p0[t], b->p1[t], b->p2[t], b->rc[t], &v[t], &dV);
        }
    return v;
}

/* ---------------------------------------------------------------- threading over systems       */
typedef int (*sys_fn)(void *job, int s);
typedef struct { sys_fn fn; void *job; int s0, s1, stride, rc; } tjob;
static void *trun(void *p)
{
    tjob *t = (tjob *)p;
    for (int s = t->s0; s < t->s1; s += t->stride) {
        int rc = t->fn(t->job, s);
        if (rc != ORC_OK) t->rc = rc;
    }
    return NULL;
}
static int for_systems(int S, int nthreads, sys_fn fn, void *job)
{
    if (nthreads < 1) nthreads = 1;
    if (nthreads > S) nthreads = S > 0 ? S : 1;
    if (nthreads > 256) nthreads = 256;
    pthread_t th[256]; tjob tj[256];
    for (int t = 0; t < nthreads; ++t) {
        tj[t].fn = fn; tj[t].job = job; tj[t].s0 = t; tj[t].s1 = S; tj[t].stride = nthreads; tj[t].rc = ORC_OK;
        if (t > 0) pthread_create(&th[t], NULL, trun, &tj[t]);
    }
    trun(&tj[0]);
    int rc = tj[0].rc;
    for (int t = 1; t < nthreads; ++t) { pthread_join(th[t], NULL); if (tj[t].rc != ORC_OK) rc = tj[t].rc; }
    return rc;
}

/* ---------------------------------------------------------------- O2 batch entry               */
typedef struct { const orc_batch *b; const double *vshift; double *E, *W, *Eabs; } efjob;
static int ef_sys(void *vj, int s)
{
    efjob *j = (efjob *)vj;
    return system_energy_forces(j->b, s, j->vshift, j->E ? j->E + s : NULL, j->W ? j->W + 9 * s : NULL,
                                j->Eabs ? j->Eabs + s : NULL);
}
int orc_energy_forces(const orc_batch *b, double *E, double *W, double *Eabs, int nthreads)
{
    double *vs = make_vshift(b);
    efjob j = { b, vs, E, W, Eabs };
    int rc = for_systems(b->n_systems, nthreads, ef_sys, &j);
    free(vs);
    return rc;
}

/* KE_s = 1/2 sum m mass_conv v^2 (O3, R17).                                                     */
static double system_kinetic(const orc_batch *b, int s)
{
    ksum k = { 0, 0 };
    for (int64_t i = b->sys_off[s]; i < b->sys_off[s + 1]; ++i) {
        const double *v = b->vel + 3 * i;
        kadd(&k, 0.5 * b->mass[i] * b->mass_conv * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
    }
    return kval(&k);
}
int orc_kinetic(const orc_batch *b, double *KE)
{
    for (int s = 0; s < b->n_systems; ++s) KE[s] = system_kinetic(b, s);
    return ORC_OK;
}

/* ---------------------------------------------------------------- O5: Philox4x32-10 + normals  */
static void mulhilo(uint32_t a, uint32_t b, uint32_t *hi, uint32_t *lo)
{
    uint64_t p = (uint64_t)a * (uint64_t)b;
    *hi = (uint32_t)(p >> 32); *lo = (uint32_t)p;
}
void orc_philox4x32_10(const uint32_t *ctr, const uint32_t *key, uint32_t *out)
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint32_t hi0, lo0, hi1, lo1;
        mulhilo(0xD2511F53u, c0, &hi0, &lo0);
        mulhilo(0xCD9E8D57u, c2, &hi1, &lo1);
        uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;   /* bumped between rounds; the 10th bump is unused */
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Box-Muller on four 32-bit words (O5, R19): u_k = (w_k + 0.5) 2^-32 in (0,1).                  */
void orc_normals_from_words(const uint32_t *w, double *xi)
{
    double u[4];
    for (int k = 0; k < 4; ++k) u[k] = ((double)w[k] + 0.5) * (1.0 / 4294967296.0);
    const double two_pi = 6.283185307179586476925286766559;
    double r0 = sqrt(-2.0 * log(u[0])), r1 = sqrt(-2.0 * log(u[2]));
    xi[0] = r0 * cos(two_pi * u[1]);
    xi[1] = r0 * sin(two_pi * u[1]);
    xi[2] = r1 * cos(two_pi * u[3]);
}

/* xi in R^3 for (seed; sys_uid, local atom index, step), purpose 0 = Langevin O-step (O5, R18). */
void orc_langevin_xi(uint64_t seed, uint32_t sys_uid, uint32_t local_idx, uint64_t step, double *xi)
{
    uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { local_idx, sys_uid, (uint32_t)(step & 0xffffffffu), (uint32_t)(step >> 32) | (0u << 24) };
    uint32_t w[4];
    orc_philox4x32_10(ctr, key, w);
    orc_normals_from_words(w, xi);
}

/* ---------------------------------------------------------------- O3 / O4: MD                  */
typedef struct {
    orc_batch *b; const double *vshift;
    int integrator; double dt, T, gamma; uint64_t seed;
    const uint32_t *sys_uid; uint64_t *step;
    int n_steps; double *E, *W, *KE, *epot_hist, *ke_hist;
} mdjob;

static int md_sys(void *vj, int s)
{
    mdjob *j = (mdjob *)vj;
    orc_batch *b = j->b;
    int S = b->n_systems;
    int64_t a0 = b->sys_off[s], a1 = b->sys_off[s + 1];
    double E, W[9];
    int rc = system_energy_forces(b, s, j->vshift, &E, W, NULL);   /* forces made current       */
    if (rc != ORC_OK) return rc;
    if (j->epot_hist) j->epot_hist[s] = E;
    if (j->ke_hist) j->ke_hist[s] = system_kinetic(b, s);
    double dt = j->dt, hdt = 0.5 * dt;
    double c1 = exp(-j->gamma * dt), c2 = sqrt(1.0 - c1 * c1);
    uint32_t uid = j->sys_uid ? j->sys_uid[s] : (uint32_t)s;
    for (int n = 0; n < j->n_steps; ++n) {
        uint64_t step = j->step ? j->step[s] : (uint64_t)n;
        for (int64_t i = a0; i < a1; ++i) {
            double im = 1.0 / (b->mass[i] * b->mass_conv);
            double *x = b->pos + 3 * i, *v = b->vel + 3 * i, *f = b->force + 3 * i;
            if (j->integrator == 0) {                /* O3 velocity Verlet: kick, drift          */
                for (int k = 0; k < 3; ++k) { v[k] = v[k] + hdt * (f[k] * im); x[k] = x[k] + dt * v[k]; }
            } else {                                 /* O4 BAOAB: B A O A                        */
                double xi[3];
                orc_langevin_xi(j->seed, uid, (uint32_t)(i - a0), step, xi);
                double sig = sqrt(b->kB * j->T * im);
                for (int k = 0; k < 3; ++k) {
                    v[k] = v[k] + hdt * (f[k] * im);
                    x[k] = x[k] + hdt * v[k];
                    v[k] = c1 * v[k] + c2 * sig * xi[k];
                    x[k] = x[k] + hdt * v[k];
                }
            }
        }
        rc = system_energy_forces(b, s, j->vshift, &E, W, NULL);
        if (rc != ORC_OK) return rc;
        for (int64_t i = a0; i < a1; ++i) {          /* final B                                  */
            double im = 1.0 / (b->mass[i] * b->mass_conv);
            double *v = b->vel + 3 * i, *f = b->force + 3 * i;
            for (int k = 0; k < 3; ++k) v[k] = v[k] + hdt * (f[k] * im);
        }
        if (j->step) j->step[s] += 1;
        if (j->epot_hist) j->epot_hist[(size_t)(n + 1) * S + s] = E;
        if (j->ke_hist) j->ke_hist[(size_t)(n + 1) * S + s] = system_kinetic(b, s);
    }
    if (j->E) j->E[s] = E;
    if (j->W) memcpy(j->W + 9 * s, W, sizeof W);
    if (j->KE) j->KE[s] = system_kinetic(b, s);
    return ORC_OK;
}

/* n_steps of O3 (integrator 0) or O4 (integrator 1) on every system.  pos, vel, force updated in
 * place (R16).  step[s] (may be NULL -> 0,1,2,...) is the system's own step counter (R18) and is
 * advanced.  epot_hist/ke_hist (may be NULL) are [(n_steps+1), S], row 0 = initial state.       */
int orc_md_run(orc_batch *b, int integrator, double dt, double T, double gamma, uint64_t seed,
               const uint32_t *sys_uid, uint64_t *step, int n_steps, double *E, double *W,
               double *KE, double *epot_hist, double *ke_hist, int nthreads)
{
    double *vs = make_vshift(b);
    mdjob j = { b, vs, integrator, dt, T, gamma, seed, sys_uid, step, n_steps, E, W, KE, epot_hist, ke_hist };
    int rc = for_systems(b->n_systems, nthreads, md_sys, &j);
    free(vs);
    return rc;
}

/* ---------------------------------------------------------------- O6: FIRE                     */
enum { FIRE_FRESH = 0, FIRE_RUNNING = 1, FIRE_CONVERGED = 2, FIRE_FAILED = 3 };
typedef struct {
    orc_batch *b; const double *vshift; const orc_fire_params *p; int n_steps;
    double *dt, *alpha; int32_t *npos, *nsteps, *status; double *E, *fmax;
} firejob;

static double max_force_norm(const orc_batch *b, int s)
{
    double m = 0.0;
    for (int64_t i = b->sys_off[s]; i < b->sys_off[s + 1]; ++i) {
        const double *f = b->force + 3 * i;
        double n = sqrt(f[0] * f[0] + f[1] * f[1] + f[2] * f[2]);
        if (n > m) m = n;
    }
    return m;
}

static int fire_sys(void *vj, int s)
{
    firejob *j = (firejob *)vj;
    orc_batch *b = j->b; const orc_fire_params *p = j->p;
    int64_t a0 = b->sys_off[s], a1 = b->sys_off[s + 1];
    double E; int rc;
    if (j->status[s] == FIRE_CONVERGED || j->status[s] == FIRE_FAILED) return ORC_OK; /* frozen */
    if (j->status[s] == FIRE_FRESH) {                 /* O6 init                                 */
        for (int64_t i = 3 * a0; i < 3 * a1; ++i) b->vel[i] = 0.0;
        j->dt[s] = p->dt_start; j->alpha[s] = p->alpha_start; j->npos[s] = 0; j->nsteps[s] = 0;
        rc = system_energy_forces(b, s, j->vshift, &E, NULL, NULL);
        if (rc != ORC_OK) return rc;
        j->E[s] = E; j->fmax[s] = max_force_norm(b, s);
        j->status[s] = (j->fmax[s] < p->f_max) ? FIRE_CONVERGED : FIRE_RUNNING;
        if (j->status[s] == FIRE_CONVERGED) return ORC_OK;
    } else {
        rc = system_energy_forces(b, s, j->vshift, &E, NULL, NULL);    /* forces made current   */
        if (rc != ORC_OK) return rc;
    }
    for (int n = 0; n < j->n_steps; ++n) {
        if (j->nsteps[s] >= p->max_steps) { j->status[s] = FIRE_FAILED; break; }
        double dt = j->dt[s], hdt = 0.5 * dt;
        for (int64_t i = a0; i < a1; ++i) {           /* (1) velocity-Verlet step with own dt    */
            double im = 1.0 / (b->mass[i] * b->mass_conv);
            double *x = b->pos + 3 * i, *v = b->vel + 3 * i, *f = b->force + 3 * i;
            for (int k = 0; k < 3; ++k) { v[k] = v[k] + hdt * (f[k] * im); x[k] = x[k] + dt * v[k]; }
        }
        rc = system_energy_forces(b, s, j->vshift, &E, NULL, NULL);
        if (rc != ORC_OK) return rc;
        for (int64_t i = a0; i < a1; ++i) {
            double im = 1.0 / (b->mass[i] * b->mass_conv);
            double *v = b->vel + 3 * i, *f = b->force + 3 * i;
            for (int k = 0; k < 3; ++k) v[k] = v[k] + hdt * (f[k] * im);
        }
        j->nsteps[s] += 1;
        j->E[s] = E; j->fmax[s] = max_force_norm(b, s);
        if (j->fmax[s] < p->f_max) { j->status[s] = FIRE_CONVERGED; break; }   /* (2) freeze      */
        ksum P = { 0, 0 }, vv = { 0, 0 }, ff = { 0, 0 };
        for (int64_t i = 3 * a0; i < 3 * a1; ++i) {   /* (3) P = F.v and the 3N-dim norms        */
            kadd(&P, b->force[i] * b->vel[i]);
            kadd(&vv, b->vel[i] * b->vel[i]);
            kadd(&ff, b->force[i] * b->force[i]);
        }
        if (kval(&P) > 0.0) {                         /* (4) mix with the alpha before update    */
            double fn = sqrt(kval(&ff)), vn = sqrt(kval(&vv)), al = j->alpha[s];
            if (fn > 0.0) {
                double cf = al * (vn / fn);
                for (int64_t i = 3 * a0; i < 3 * a1; ++i)
                    b->vel[i] = (1.0 - al) * b->vel[i] + cf * b->force[i];
            }
            j->npos[s] += 1;
            if (j->npos[s] > p->n_min) {
                double nd = j->dt[s] * p->f_inc;
                j->dt[s] = nd < p->dt_max ? nd : p->dt_max;
                j->alpha[s] = j->alpha[s] * p->f_alpha;
            }
        } else {                                      /* (5) uphill: stop, halve dt, reset       */
            for (int64_t i = 3 * a0; i < 3 * a1; ++i) b->vel[i] = 0.0;
            j->dt[s] = j->dt[s] * p->f_dec; j->alpha[s] = p->alpha_start; j->npos[s] = 0;
        }
    }
    return ORC_OK;
}

/* Up to n_steps FIRE steps (O6) on every system that is not frozen.  Per-system state arrays
 * dt, alpha, npos, nsteps, status are in/out (status FIRE_FRESH triggers initialisation).       */
int orc_fire_run(orc_batch *b, const orc_fire_params *p, int n_steps, double *dt, double *alpha,
                 int32_t *npos, int32_t *nsteps, int32_t *status, double *E, double *fmax,
                 int nthreads)
{
    double *vs = make_vshift(b);
    firejob j = { b, vs, p, n_steps, dt, alpha, npos, nsteps, status, E, fmax };
    int rc = for_systems(b->n_systems, nthreads, fire_sys, &j);
    free(vs);
    return rc;
}
