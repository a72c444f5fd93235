/*
 * ts_repack.cu -- ragged in-flight replacement (kernel K12; "removes
 * converged systems and samples new systems from the stream until memory is full", :96 Fig. 3: systems
 * of different sizes share one batch).  ts_repack_systems re-lays the SoA state: the batch becomes the
 * kept systems, in the caller's order, followed by the fresh ones, whatever their sizes; the per-system
 * state of the kept systems (FIRE scalars, step counters, uids, cells) moves with them.
 *
 * Device side: two gather kernels through workspace regions that the next neighbour build overwrites
 * anyway (xref, pos4, spos).  Host side: the per-system scalars make one round trip (a few bytes per
 * system; the call synchronises, as a swap does).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "ts_internal.cuh"

struct RepackSys { int new_off, n, src_off, from_fresh; };

/* block k gathers the atoms of new system k into the temporaries */
template <typename T>
__global__ void k_repack_gather(DevState d, const RepackSys *tab, T *tpos, T *tvel, T *tmass, int *ttype,
                                const T *fpos, const T *fvel, const T *fmass, const int *ftype)
{
    const RepackSys r = tab[blockIdx.x];
    const T *spos = r.from_fresh ? fpos : (const T *)d.pos, *svel = r.from_fresh ? fvel : (const T *)d.vel;
    const T *smass = r.from_fresh ? fmass : (const T *)d.mass;
    const int *stype = r.from_fresh ? ftype : d.type;
    for (int t = threadIdx.x; t < 3 * r.n; t += blockDim.x) {
        tpos[3 * (size_t)r.new_off + t] = spos[3 * (size_t)r.src_off + t];
        tvel[3 * (size_t)r.new_off + t] = svel ? svel[3 * (size_t)r.src_off + t] : (T)0;
    }
    for (int t = threadIdx.x; t < r.n; t += blockDim.x) {
        tmass[r.new_off + t] = smass[r.src_off + t];
        ttype[r.new_off + t] = stype[r.src_off + t];
    }
}

/* block k writes new system k into the live arrays */
template <typename T>
__global__ void k_repack_scatter(DevState d, const RepackSys *tab, int S_new, const T *tpos, const T *tvel, const T *tmass,
                                 const int *ttype)
{
    const RepackSys r = tab[blockIdx.x];
    T *pos = (T *)d.pos, *vel = (T *)d.vel, *mass = (T *)d.mass;
    int *type = (int *)d.type, *sysidx = (int *)d.sysidx;
    for (int t = threadIdx.x; t < 3 * r.n; t += blockDim.x) {
        pos[3 * (size_t)r.new_off + t] = tpos[3 * (size_t)r.new_off + t];
        vel[3 * (size_t)r.new_off + t] = tvel[3 * (size_t)r.new_off + t];
    }
    for (int t = threadIdx.x; t < r.n; t += blockDim.x) {
        mass[r.new_off + t] = tmass[r.new_off + t];
        type[r.new_off + t] = ttype[r.new_off + t];
        sysidx[r.new_off + t] = (int)blockIdx.x;
    }
    if (threadIdx.x == 0) {
        d.sysoff[blockIdx.x] = r.new_off;
        if ((int)blockIdx.x == S_new - 1) d.sysoff[S_new] = r.new_off + r.n;
    }
}

template <typename V>
static bool pull(std::vector<V> &h, const V *dev, size_t n)
{
    h.resize(n);
    return n == 0 || cudaMemcpy(h.data(), dev, sizeof(V) * n, cudaMemcpyDeviceToHost) == cudaSuccess;
}
template <typename V>
static bool push(const std::vector<V> &h, V *dev)
{
    return h.empty() || cudaMemcpy(dev, h.data(), sizeof(V) * h.size(), cudaMemcpyHostToDevice) == cudaSuccess;
}
template <typename V>
static std::vector<V> permute(const std::vector<V> &old, const int32_t *keep, int n_keep, int n_fresh, V fresh_value, int per = 1)
{
    std::vector<V> out((size_t)(n_keep + n_fresh) * per, fresh_value);
    for (int k = 0; k < n_keep; ++k)
        for (int c = 0; c < per; ++c) out[(size_t)k * per + c] = old[(size_t)keep[k] * per + c];
    return out;
}

extern "C" ts_status ts_repack_systems(ts_state *st, const int32_t *keep, int32_t n_keep, const ts_state_desc *fresh,
                                       const int32_t *fresh_n_atoms, void *stream)
{
    if (!st) return TS_ERR_INVALID_ARG;
    if (st->seen_flags) return TS_ERR_STICKY;
    const int n_fresh = fresh ? fresh->n_systems : 0;
    if (n_keep < 0 || n_fresh < 0 || n_keep + n_fresh < 1 || (n_keep > 0 && !keep) || (n_fresh > 0 && !fresh_n_atoms))
        return TS_ERR_INVALID_ARG;
    if (n_fresh > 0 && (!fresh->pos || !fresh->mass || !fresh->type || !fresh->cell || fresh->dtype != st->d.dtype))
        return TS_ERR_INVALID_ARG;
    cudaStream_t q = (cudaStream_t)stream;
    DevState &d = st->d;
    const int S_old = d.S, S_new = n_keep + n_fresh;
    const size_t w = d.dtype == TS_F32 ? 4 : 8;
    if (S_new > st->S_cap) return TS_ERR_WORKSPACE_TOO_SMALL;

    /* the new layout */
    std::vector<RepackSys> tab((size_t)S_new);
    std::vector<char> seen((size_t)S_old, 0);
    long long off = 0, foff = 0;
    for (int k = 0; k < S_new; ++k) {
        RepackSys r;
        if (k < n_keep) {
            const int s = keep[k];
            if (s < 0 || s >= S_old || seen[(size_t)s]) return TS_ERR_INVALID_ARG;
            seen[(size_t)s] = 1;
            r.n = st->h_sysoff[s + 1] - st->h_sysoff[s]; r.src_off = st->h_sysoff[s]; r.from_fresh = 0;
        } else {
            r.n = fresh_n_atoms[k - n_keep];
            if (r.n < 1 || r.n > TS_MAX_SYS_ATOMS) return TS_ERR_INVALID_ARG;
            r.src_off = (int)foff; r.from_fresh = 1;
            foff += r.n;
        }
        r.new_off = (int)off;
        off += r.n;
        tab[(size_t)k] = r;
    }
    if (n_fresh > 0 && foff != fresh->n_atoms) return TS_ERR_INVALID_ARG;
    if (off > st->N_cap) return TS_ERR_WORKSPACE_TOO_SMALL;

    TS_CUDA_OK(st, cudaStreamSynchronize(q));
    /* per-system state: one host round trip */
    std::vector<double> f_dt, f_alpha;
    std::vector<int> f_npos, f_nsteps, f_status, sys_active;
    std::vector<unsigned long long> sys_step;
    std::vector<unsigned> uid, fuid;
    std::vector<char> cell, fcell;
    if (!pull(f_dt, d.f_dt, (size_t)S_old) || !pull(f_alpha, d.f_alpha, (size_t)S_old) || !pull(f_npos, d.f_npos, (size_t)S_old) ||
        !pull(f_nsteps, d.f_nsteps, (size_t)S_old) || !pull(f_status, d.f_status, (size_t)S_old) ||
        !pull(sys_active, d.sys_active, (size_t)S_old) || !pull(sys_step, d.sys_step, (size_t)S_old) ||
        !pull(uid, d.uid_own, (size_t)S_old) || !pull(cell, (const char *)d.cell, 9 * w * (size_t)S_old))
        return TS_ERR_CUDA;
    if (n_fresh > 0) {
        if (!pull(fcell, (const char *)fresh->cell, 9 * w * (size_t)n_fresh)) return TS_ERR_CUDA;
        if (fresh->sys_uid && !pull(fuid, (const unsigned *)fresh->sys_uid, (size_t)n_fresh)) return TS_ERR_CUDA;
    }
    std::vector<double> n_dt = permute(f_dt, keep, n_keep, n_fresh, 0.0), n_alpha = permute(f_alpha, keep, n_keep, n_fresh, 0.0);
    std::vector<int> n_npos = permute(f_npos, keep, n_keep, n_fresh, 0), n_nsteps = permute(f_nsteps, keep, n_keep, n_fresh, 0);
    std::vector<int> n_status = permute(f_status, keep, n_keep, n_fresh, (int)TS_FIRE_FRESH);
    std::vector<int> n_active = permute(sys_active, keep, n_keep, n_fresh, 1);
    std::vector<unsigned long long> n_step = permute(sys_step, keep, n_keep, n_fresh, 0ull);
    std::vector<unsigned> n_uid = permute(uid, keep, n_keep, n_fresh, 0u);
    std::vector<char> n_cell = permute(cell, keep, n_keep, n_fresh, (char)0, (int)(9 * w));
    for (int k = 0; k < n_fresh; ++k) {
        n_uid[(size_t)(n_keep + k)] = fresh->sys_uid ? fuid[(size_t)k] : (unsigned)(n_keep + k);
        memcpy(n_cell.data() + 9 * w * (size_t)(n_keep + k), fcell.data() + 9 * w * (size_t)k, 9 * w);
    }
    /* pair capacity of the new batch (the paper's n_atoms_x_density scaler, as at create) */
    std::vector<long long> base((size_t)S_new + 1, 0);
    for (int k = 0; k < S_new; ++k) {
        double h[9];
        for (int c = 0; c < 9; ++c)
            h[c] = d.dtype == TS_F32 ? (double)((const float *)n_cell.data())[9 * (size_t)k + c] : ((const double *)n_cell.data())[9 * (size_t)k + c];
        const double det = h[0] * (h[4] * h[8] - h[5] * h[7]) + h[1] * (h[5] * h[6] - h[3] * h[8]) + h[2] * (h[3] * h[7] - h[4] * h[6]);
        if (!(fabs(det) > 0.0)) return TS_ERR_INVALID_ARG;
        base[(size_t)k + 1] = base[(size_t)k] + ts_system_pair_capacity(tab[(size_t)k].n, fabs(det), d.r_list, st->nbr.slack);
    }
    if (base.back() > d.nbr_cap) return TS_ERR_WORKSPACE_TOO_SMALL;

    /* atoms: gather into the temporaries, then back (xref: positions, pos4: velocities, spos: masses, types, table) */
    char *sp = (char *)d.spos;
    void *tpos = d.xref, *tvel = d.pos4, *tmass = sp;
    int *ttype = (int *)(sp + 8 * (size_t)st->N_cap);
    RepackSys *dtab = (RepackSys *)(sp + 12 * (size_t)st->N_cap);
    TS_CUDA_OK(st, cudaMemcpyAsync(dtab, tab.data(), sizeof(RepackSys) * tab.size(), cudaMemcpyHostToDevice, q));
    if (d.dtype == TS_F32) {
        k_repack_gather<float><<<S_new, 256, 0, q>>>(d, dtab, (float *)tpos, (float *)tvel, (float *)tmass, ttype,
                                                    n_fresh ? (const float *)fresh->pos : nullptr, n_fresh ? (const float *)fresh->vel : nullptr,
                                                    n_fresh ? (const float *)fresh->mass : nullptr, n_fresh ? fresh->type : nullptr);
        k_repack_scatter<float><<<S_new, 256, 0, q>>>(d, dtab, S_new, (const float *)tpos, (const float *)tvel, (const float *)tmass, ttype);
    } else {
        k_repack_gather<double><<<S_new, 256, 0, q>>>(d, dtab, (double *)tpos, (double *)tvel, (double *)tmass, ttype,
                                                     n_fresh ? (const double *)fresh->pos : nullptr, n_fresh ? (const double *)fresh->vel : nullptr,
                                                     n_fresh ? (const double *)fresh->mass : nullptr, n_fresh ? fresh->type : nullptr);
        k_repack_scatter<double><<<S_new, 256, 0, q>>>(d, dtab, S_new, (const double *)tpos, (const double *)tvel, (const double *)tmass, ttype);
    }
    st->launches += 2;
    TS_CUDA_OK(st, cudaStreamSynchronize(q));               /* the table must outlive the kernels; the scalars follow */
    if (!push(n_dt, d.f_dt) || !push(n_alpha, d.f_alpha) || !push(n_npos, d.f_npos) || !push(n_nsteps, d.f_nsteps) ||
        !push(n_status, d.f_status) || !push(n_active, d.sys_active) || !push(n_step, d.sys_step) || !push(n_uid, d.uid_own) ||
        !push(n_cell, (char *)d.cell) || !push(base, d.nbr_base))
        return TS_ERR_CUDA;

    /* host view of the new batch */
    d.N = off; d.S = S_new;
    st->desc.n_atoms = off; st->desc.n_systems = S_new;
    for (int k = 0; k < S_new; ++k) st->h_sysoff[k] = tab[(size_t)k].new_off;
    st->h_sysoff[S_new] = (int)off;
    launch_geometry(st, 0, S_new, nullptr, q);
    resident_invalidate(st);
    st->list_built = false;
    st->forces_current = false;
    TS_CUDA_OK(st, cudaStreamSynchronize(q));
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { ts_set_error(st, "repack failed: %s", cudaGetErrorString(e)); return TS_ERR_CUDA; }
    return TS_OK;
}

extern "C" ts_status ts_estimate_system_pairs(int64_t n_atoms, double volume, double r_list, double slack, int64_t *out_pairs)
{
    if (!out_pairs || n_atoms < 1 || !(volume > 0.0) || !(r_list > 0.0)) return TS_ERR_INVALID_ARG;
    *out_pairs = ts_system_pair_capacity(n_atoms, volume, r_list, slack);
    return TS_OK;
}

extern "C" ts_status ts_get_capacity(const ts_state *st, int64_t *n_atoms, int32_t *n_systems, int64_t *n_pairs)
{
    if (!st) return TS_ERR_INVALID_ARG;
    if (n_atoms) *n_atoms = st->N_cap;
    if (n_systems) *n_systems = st->S_cap;
    if (n_pairs) *n_pairs = st->d.nbr_cap;
    return TS_OK;
}
