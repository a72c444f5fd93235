/*
 * ts_api.cu -- the C ABI of libts (include/ts.h): argument checks, workspace carving, the memory
 * estimate, and the host-side sequencing of the kernels.  No device memory is
 * allocated here: every device byte is the caller's (boundary arrays + workspace blob).
 */
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "ts_internal.cuh"

void ts_set_error(ts_state *st, const char *fmt, ...)
{
    if (!st) return;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(st->err, sizeof st->err, fmt, ap);
    va_end(ap);
}

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

TsLayout ts_layout(long long N, int S, long long nbr_cap, int dtype, int n_types)
{
    TsLayout L;
    size_t o = 0;
    size_t w = dtype == TS_F32 ? 4 : 8;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    L.status = take(sizeof(DevStatus));
    L.sysoff = take(sizeof(int) * (size_t)(S + 1));
    L.geom = take(sizeof(SysGeom) * (size_t)S);
    L.hT = take(w * 9 * (size_t)S);
    L.nbr_base = take(sizeof(long long) * (size_t)(S + 1));
    L.nbr_len = take(sizeof(long long) * (size_t)S);
    L.f_dt = take(8 * (size_t)S);
    L.f_alpha = take(8 * (size_t)S);
    L.f_npos = take(4 * (size_t)S);
    L.f_nsteps = take(4 * (size_t)S);
    L.f_status = take(4 * (size_t)S);
    L.f_acc = take(8 * 4 * (size_t)S);
    L.sys_active = take(4 * (size_t)S);
    L.sys_rebuild = take(4 * (size_t)S);
    L.sys_step = take(8 * (size_t)S);
    L.uid_own = take(4 * (size_t)S);
    L.sys_engine = take(4 * (size_t)S);
    L.res_list = take(4 * (size_t)S);
    L.res_saved = take(4 * (size_t)S);
    L.red_slots = take(64 * ((size_t)N / 4 + (size_t)S + 2));
    L.scratch = take(4 * (2 * (size_t)S + 8));
    L.pot = take(sizeof(PotEntry<double>) * (size_t)n_types * n_types);
    L.pos4 = take(4 * w * (size_t)N);
    L.spos = take(sizeof(double4) * (size_t)N);
    L.xref = take(3 * w * (size_t)N);
    L.cell_count = take(4 * (size_t)(N + S + 1));
    L.cell_start = take(4 * (size_t)(N + S + 1));
    L.atom_cell = take(4 * (size_t)N);
    L.atom_rank = take(4 * (size_t)N);
    L.atom_wrap = take(4 * (size_t)N);
    L.nbr_cnt = take(4 * (size_t)N);
    L.nbr_off = take(8 * (size_t)N);
    L.nbr = take(4 * (size_t)nbr_cap);
    L.total = o;
    return L;
}

/* Pair slots reserved for a system of n atoms in volume vol: the paper's n_atoms_x_density
 * scaler (section 3) with a known coefficient: n * rho * 4/3 pi r_list^3 * slack. */
long long ts_system_pair_capacity(long long n, double vol, double r_list, double slack)
{
    if (slack < 1.0) slack = 1.25;
    double nbar = (double)n / vol * (4.0 / 3.0) * M_PI * r_list * r_list * r_list;
    double c = (double)n * (nbar * slack + 8.0);
    return (long long)ceil(c / 32.0) * 32;
}

static size_t per_atom_workspace_bytes(int dtype)
{
    size_t w = dtype == TS_F32 ? 4 : 8;
    return 4 * w + sizeof(double4) + 3 * w + 4 * 2 /* cell_count, cell_start */ + 4 * 4 + 8 + 16 /* red_slots: 64 B per 4 atoms */;
}

static double max_rc(const ts_potential *pot)
{
    double m = 0.0;
    for (int t = 0; t < pot->n_types * pot->n_types; ++t) m = pot->rc[t] > m ? pot->rc[t] : m;
    return m;
}

extern "C" ts_status ts_estimate_system_bytes(int64_t n_atoms, double volume, double r_list, double slack,
                                              int32_t dtype, size_t *out_bytes)
{
    if (!out_bytes || n_atoms < 1 || !(volume > 0.0) || !(r_list > 0.0) || (dtype != TS_F32 && dtype != TS_F64))
        return TS_ERR_INVALID_ARG;
    size_t w = dtype == TS_F32 ? 4 : 8;
    size_t boundary = (size_t)n_atoms * (3 * 3 * w + w + 4 + 4) + 9 * w + 8 * 11 + 4;
    size_t per_sys = sizeof(SysGeom) + 9 * w + 8 * 2 + 8 * 2 + 4 * 8 /* incl. sys_rebuild, sys_engine, res_list, res_saved */ + 64 /* red_slots */ + 32 + 8 + 4 + 8 + 4 * 2 /* cell slots */;
    size_t ws = (size_t)n_atoms * per_atom_workspace_bytes(dtype) + per_sys +
                4 * (size_t)ts_system_pair_capacity(n_atoms, volume, r_list, slack);
    *out_bytes = boundary + ws;
    return TS_OK;
}

static bool desc_ok(const ts_state_desc *d, const ts_potential *pot, const ts_nbr_params *nbr)
{
    if (!d || !pot || !nbr) return false;
    if (d->n_atoms < 1 || d->n_atoms > 2000000000ll || d->n_systems < 1 || d->n_systems > d->n_atoms) return false;
    if (d->dtype != TS_F32 && d->dtype != TS_F64) return false;
    if (!d->pos || !d->vel || !d->force || !d->mass || !d->type || !d->system_idx || !d->cell) return false;
    if (!d->energy || !d->virial || !d->kinetic) return false;
    if (pot->kind < TS_LJ || pot->kind > TS_SOFT_SPHERE) return false;
    if (pot->n_types < 1 || pot->n_types > TS_MAX_TYPES || !pot->p0 || !pot->p1 || !pot->p2 || !pot->rc) return false;
    if (!(nbr->skin >= 0.0) || !(max_rc(pot) > 0.0)) return false;
    if (!(d->units.mass_conv > 0.0)) return false;
    return true;
}

/* Reads system_idx and cells from the device; fills sysoff [S+1] and nbr_base [S+1]. */
static ts_status scan_batch(const ts_state_desc *d, const ts_potential *pot, const ts_nbr_params *nbr,
                            std::vector<int> &sysoff, std::vector<long long> &nbr_base)
{
    long long N = d->n_atoms;
    int S = d->n_systems;
    std::vector<int> idx((size_t)N);
    if (cudaMemcpy(idx.data(), d->system_idx, sizeof(int) * (size_t)N, cudaMemcpyDeviceToHost) != cudaSuccess)
        return TS_ERR_CUDA;
    sysoff.assign((size_t)S + 1, 0);
    int prev = 0;
    if (idx[0] != 0) return TS_ERR_INVALID_ARG;
    for (long long i = 0; i < N; ++i) {
        int s = idx[(size_t)i];
        if (s < prev || s > prev + 1 || s >= S) return TS_ERR_INVALID_ARG;   /* non-decreasing, no empty system */
        prev = s;
        sysoff[(size_t)s + 1] += 1;
    }
    if (prev != S - 1) return TS_ERR_INVALID_ARG;
    for (int s = 0; s < S; ++s) {
        if (sysoff[(size_t)s + 1] > TS_MAX_SYS_ATOMS) return TS_ERR_UNSUPPORTED;
        sysoff[(size_t)s + 1] += sysoff[(size_t)s];
    }
    size_t w = d->dtype == TS_F32 ? 4 : 8;
    std::vector<char> raw(9 * w * (size_t)S);
    if (cudaMemcpy(raw.data(), d->cell, raw.size(), cudaMemcpyDeviceToHost) != cudaSuccess) return TS_ERR_CUDA;
    double r_list = max_rc(pot) + nbr->skin;
    nbr_base.assign((size_t)S + 1, 0);
    for (int s = 0; s < S; ++s) {
        double h[9];
        for (int k = 0; k < 9; ++k)
            h[k] = d->dtype == TS_F32 ? (double)((const float *)raw.data())[9 * (size_t)s + k]
                                      : ((const double *)raw.data())[9 * (size_t)s + k];
        double det = h[0] * (h[4] * h[8] - h[5] * h[7]) + h[1] * (h[5] * h[6] - h[3] * h[8]) +
                     h[2] * (h[3] * h[7] - h[4] * h[6]);
        if (!(fabs(det) > 0.0)) return TS_ERR_INVALID_ARG;
        long long n = sysoff[(size_t)s + 1] - sysoff[(size_t)s];
        nbr_base[(size_t)s + 1] = nbr_base[(size_t)s] + ts_system_pair_capacity(n, fabs(det), r_list, nbr->slack);
    }
    return TS_OK;
}

extern "C" ts_status ts_workspace_bytes(const ts_state_desc *desc, const ts_potential *pot,
                                        const ts_nbr_params *nbr, size_t *out_bytes)
{
    if (!desc_ok(desc, pot, nbr) || !out_bytes) return TS_ERR_INVALID_ARG;
    std::vector<int> sysoff;
    std::vector<long long> base;
    ts_status rc = scan_batch(desc, pot, nbr, sysoff, base);
    if (rc != TS_OK) return rc;
    *out_bytes = ts_layout(desc->n_atoms, desc->n_systems, base.back(), desc->dtype, pot->n_types).total;
    return TS_OK;
}

template <typename T>
static void fill_pot(const ts_potential *pot, std::vector<char> &buf)
{
    int nt = pot->n_types;
    buf.resize(sizeof(PotEntry<T>) * (size_t)nt * nt);
    PotEntry<T> *e = (PotEntry<T> *)buf.data();
    for (int t = 0; t < nt * nt; ++t) {
        double p0 = pot->p0[t], p1 = pot->p1[t], p2 = pot->p2[t], rc = pot->rc[t];
        double c0 = 0, c1 = 0, c2 = 0, vs = 0;
        if (pot->kind == TS_LJ) {
            double s6 = pow(p1, 6.0);
            c0 = 4.0 * p0 * s6 * s6; c1 = 4.0 * p0 * s6;
            double ir6 = 1.0 / pow(rc, 6.0);
            vs = c0 * ir6 * ir6 - c1 * ir6;
        } else if (pot->kind == TS_MORSE) {
            c0 = 2.0 * p0 * p1;
            double ex = exp(-p1 * (rc - p2));
            vs = p0 * ((1.0 - ex) * (1.0 - ex) - 1.0);
        } else {
            c0 = p0 / p2; c1 = p0 / p1; c2 = 1.0 / p1;
            double u = 1.0 - rc / p1;
            vs = u > 0.0 ? c0 * pow(u, p2) : 0.0;
        }
        if (!pot->shift_energy) vs = 0.0;
        e[t].p0 = (T)p0; e[t].p1 = (T)p1; e[t].p2 = (T)p2; e[t].rc2 = (T)(rc * rc); e[t].vshift = (T)vs;
        e[t].c0 = (T)c0; e[t].c1 = (T)c1; e[t].c2 = (T)c2;
    }
}

extern "C" ts_status ts_state_create(const ts_state_desc *desc, const ts_potential *pot,
                                     const ts_nbr_params *nbr, void *workspace, size_t workspace_bytes,
                                     ts_state **out)
{
    if (!out) return TS_ERR_INVALID_ARG;
    *out = nullptr;
    if (!desc_ok(desc, pot, nbr) || !workspace || ((uintptr_t)workspace & 255)) return TS_ERR_INVALID_ARG;
    std::vector<int> sysoff;
    std::vector<long long> base;
    ts_status rc = scan_batch(desc, pot, nbr, sysoff, base);
    if (rc != TS_OK) return rc;
    long long N = desc->n_atoms;
    int S = desc->n_systems;
    TsLayout L = ts_layout(N, S, base.back(), desc->dtype, pot->n_types);
    if (workspace_bytes < L.total) return TS_ERR_WORKSPACE_TOO_SMALL;

    ts_state *st = (ts_state *)calloc(1, sizeof(ts_state));
    if (!st) return TS_ERR_INVALID_ARG;
    st->desc = *desc;
    st->nbr = *nbr;
    st->engine = 1;
    st->N_cap = N; st->S_cap = S;
    st->h_sysoff = (int *)malloc(sizeof(int) * (size_t)(S + 1));
    memcpy(st->h_sysoff, sysoff.data(), sizeof(int) * (size_t)(S + 1));
    char *ws = (char *)workspace;
    DevState &d = st->d;
    d.N = N; d.S = S; d.dtype = desc->dtype;
    d.kind = pot->kind; d.n_types = pot->n_types; d.shift_energy = pot->shift_energy;
    d.mass_conv = desc->units.mass_conv; d.kB = desc->units.kB;
    d.r_list = max_rc(pot) + nbr->skin; d.r_list2 = d.r_list * d.r_list;
    d.half_skin2 = 0.25 * nbr->skin * nbr->skin;
    d.pos = desc->pos; d.vel = desc->vel; d.force = desc->force; d.mass = desc->mass;
    d.type = desc->type; d.sysidx = desc->system_idx; d.cell = desc->cell;
    d.energy = desc->energy; d.virial = desc->virial; d.kinetic = desc->kinetic; d.uid = desc->sys_uid;
    d.status = (DevStatus *)(ws + L.status);
    d.sysoff = (int *)(ws + L.sysoff); d.geom = (SysGeom *)(ws + L.geom); d.hT = ws + L.hT;
    d.nbr_base = (long long *)(ws + L.nbr_base); d.nbr_len = (long long *)(ws + L.nbr_len);
    d.f_dt = (double *)(ws + L.f_dt); d.f_alpha = (double *)(ws + L.f_alpha);
    d.f_npos = (int *)(ws + L.f_npos); d.f_nsteps = (int *)(ws + L.f_nsteps); d.f_status = (int *)(ws + L.f_status);
    d.f_acc = (double *)(ws + L.f_acc); d.sys_active = (int *)(ws + L.sys_active); d.sys_rebuild = (int *)(ws + L.sys_rebuild);
    d.sys_step = (unsigned long long *)(ws + L.sys_step); d.uid_own = (unsigned int *)(ws + L.uid_own);
    d.sys_engine = (int *)(ws + L.sys_engine); d.res_list = (int *)(ws + L.res_list); d.mixed = 0;
    d.res_saved = (int *)(ws + L.res_saved);
    d.red_slots = (double *)(ws + L.red_slots);
    d.scratch = (int *)(ws + L.scratch); d.pot = ws + L.pot;
    d.pos4 = ws + L.pos4; d.spos = (double4 *)(ws + L.spos); d.xref = ws + L.xref;
    d.cell_count = (int *)(ws + L.cell_count); d.cell_start = (int *)(ws + L.cell_start);
    d.atom_cell = (int *)(ws + L.atom_cell); d.atom_rank = (int *)(ws + L.atom_rank); d.atom_wrap = (int *)(ws + L.atom_wrap);
    d.nbr_cnt = (int *)(ws + L.nbr_cnt); d.nbr_off = (long long *)(ws + L.nbr_off);
    d.nbr = (unsigned int *)(ws + L.nbr); d.nbr_cap = base.back();

#define CREATE_OK(call)                                                                   \
    do {                                                                                  \
        if ((call) != cudaSuccess) { free(st->h_sysoff); free(st); return TS_ERR_CUDA; }  \
    } while (0)
    /* everything up to the per-pair region starts zeroed (FIRE status FRESH = 0, steps 0, flags 0) */
    CREATE_OK(cudaMemset(ws, 0, L.nbr));
    CREATE_OK(cudaMemcpy(d.sysoff, sysoff.data(), sizeof(int) * (size_t)(S + 1), cudaMemcpyHostToDevice));
    CREATE_OK(cudaMemcpy(d.nbr_base, base.data(), sizeof(long long) * (size_t)(S + 1), cudaMemcpyHostToDevice));
    std::vector<char> pbuf;
    if (desc->dtype == TS_F32) fill_pot<float>(pot, pbuf); else fill_pot<double>(pot, pbuf);
    CREATE_OK(cudaMemcpy(d.pot, pbuf.data(), pbuf.size(), cudaMemcpyHostToDevice));
    if (desc->sys_uid) {
        CREATE_OK(cudaMemcpy(d.uid_own, desc->sys_uid, sizeof(unsigned) * (size_t)S, cudaMemcpyDeviceToDevice));
    } else {
        std::vector<unsigned> iota((size_t)S);
        for (int s = 0; s < S; ++s) iota[(size_t)s] = (unsigned)s;
        CREATE_OK(cudaMemcpy(d.uid_own, iota.data(), sizeof(unsigned) * (size_t)S, cudaMemcpyHostToDevice));
    }
    launch_geometry(st, 0, S, nullptr, 0);
    CREATE_OK(cudaDeviceSynchronize());
    DevStatus hs;
    CREATE_OK(cudaMemcpy(&hs, d.status, sizeof hs, cudaMemcpyDeviceToHost));
    if (hs.flags & TS_FLAG_BAD_CELL) {
        free(st->h_sysoff); free(st);
        return TS_ERR_INVALID_ARG;
    }
#undef CREATE_OK
    *out = st;
    return TS_OK;
}

extern "C" ts_status ts_state_destroy(ts_state *st)
{
    if (!st) return TS_ERR_INVALID_ARG;
    resident_free(st);
    free(st->h_sysoff);
    free(st);
    return TS_OK;
}
