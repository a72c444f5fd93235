/*
 * ts_integrate.cu -- per-atom update kernels of the general (multi-kernel) engine:
 *   velocity Verlet, Langevin BAOAB with in-kernel Philox4x32-10 + Box-Muller
 *   (O4, O5, row a7), FIRE with per-system scalars and convergence (O6, row a8), the Verlet-skin
 *   check (row a4, R12) fused into every kernel that moves atoms, and the in-flight swap copy.
 */
#include "ts_internal.cuh"
#include "ts_rng.cuh"

/* x~ = x - wrap.h -> pos4, and the skin test |x - x_ref|^2 > (skin/2)^2 (strict, R12). */
template <typename T>
__device__ __forceinline__ void publish_pos(const DevState &d, long long i, int s, T x0, T x1, T x2)
{
    typedef typename Vec4<T>::type V4;
    const T *h = (const T *)d.hT + 9 * (size_t)s;
    int w0, w1, w2;
    ts_unpack_wrap(d.atom_wrap[i], w0, w1, w2);
    T f0 = (T)w0, f1 = (T)w1, f2 = (T)w2;
    V4 q;
    q.x = x0 - (f0 * h[0] + f1 * h[3] + f2 * h[6]);
    q.y = x1 - (f0 * h[1] + f1 * h[4] + f2 * h[7]);
    q.z = x2 - (f0 * h[2] + f1 * h[5] + f2 * h[8]);
    int ty = d.type[i];
    if (sizeof(T) == 4) q.w = (T)__int_as_float(ty); else q.w = (T)__longlong_as_double((long long)ty);
    ((V4 *)d.pos4)[i] = q;
    const T *xr = (const T *)d.xref + 3 * i;
    T a = x0 - xr[0], b = x1 - xr[1], c = x2 - xr[2];
    if ((double)(a * a + b * b + c * c) > d.half_skin2) { d.status->need_rebuild = 1u; d.sys_rebuild[s] = 1; }   /* only this system is rebuilt (R12) */
}

template <typename T>
__global__ void k_import(DevState d)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    const int s = d.sysidx[i];
    if (ts_skip(d, s)) return;
    const T *x = (const T *)d.pos + 3 * i;
    publish_pos<T>(d, i, s, x[0], x[1], x[2]);
}

template <typename T>
__global__ void k_md_pre(DevState d, MdConst c)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    int s = d.sysidx[i];
    if (ts_skip(d, s)) return;
    T *x = (T *)d.pos + 3 * i, *v = (T *)d.vel + 3 * i;
    const T *f = (const T *)d.force + 3 * i;
    T im = (T)1 / (((const T *)d.mass)[i] * (T)d.mass_conv);
    T hdt = (T)c.hdt, dt = (T)c.dt;
    T xx[3] = { x[0], x[1], x[2] }, vv[3] = { v[0], v[1], v[2] };
    if (c.integrator == TS_NVE) {
#pragma unroll
        for (int k = 0; k < 3; ++k) { vv[k] = vv[k] + hdt * (f[k] * im); xx[k] = xx[k] + dt * vv[k]; }
    } else {
        unsigned long long step = d.sys_step[s];
        unsigned w[4];
        philox4x32_10((unsigned)(i - d.sysoff[s]), d.uid_own[s], (unsigned)(step & 0xffffffffull),
                      (unsigned)(step >> 32), c.key0, c.key1, w);
        T xi[3];
        normals3(w, xi);
        T sig = sizeof(T) == 4 ? (T)sqrtf((float)((T)c.kT * im)) : (T)sqrt((double)((T)c.kT * im));
        T c1 = (T)c.c1, c2 = (T)c.c2;                /* sig = sqrt(kB T / (m mass_conv)) */
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            vv[k] = vv[k] + hdt * (f[k] * im);
            xx[k] = xx[k] + hdt * vv[k];
            vv[k] = c1 * vv[k] + c2 * sig * xi[k];
            xx[k] = xx[k] + hdt * vv[k];
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) { x[k] = xx[k]; v[k] = vv[k]; }
    publish_pos<T>(d, i, s, xx[0], xx[1], xx[2]);
}

/* partial sums of one double per system (ts_sys_store; k_sum_kinetic adds them); every lane of the warp calls */
__device__ __forceinline__ void seg_store(const DevState &d, int s, bool act, double val)
{
    const double part[1] = { val };
    ts_sys_store<1, 1>(d, act ? s : -1, part);
}

template <typename T>
__global__ void k_md_post(DevState d, MdConst c, int want_ke)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    bool valid = i < d.N;
    int s = 0;
    double ke = 0.0;
    if (valid) {
        s = d.sysidx[i];
        valid = !ts_skip(d, s);
    }
    if (valid) {
        T *v = (T *)d.vel + 3 * i;
        const T *f = (const T *)d.force + 3 * i;
        T m = ((const T *)d.mass)[i];
        T im = (T)1 / (m * (T)d.mass_conv);
        T hdt = (T)c.hdt;
        T v0 = v[0] + hdt * (f[0] * im), v1 = v[1] + hdt * (f[1] * im), v2 = v[2] + hdt * (f[2] * im);
        v[0] = v0; v[1] = v1; v[2] = v2;
        ke = 0.5 * (double)m * d.mass_conv * ((double)v0 * (double)v0 + (double)v1 * (double)v1 + (double)v2 * (double)v2);
        if (i == d.sysoff[s]) d.sys_step[s] += 1ull;
    }
    if (want_ke) seg_store(d, s, valid, ke);
}

template <typename T>
__global__ void k_kinetic(DevState d)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    bool valid = i < d.N;
    int s = 0;
    double ke = 0.0;
    if (valid) {
        s = d.sysidx[i];
        valid = !ts_skip(d, s);
    }
    if (valid) {
        const T *v = (const T *)d.vel + 3 * i;
        double m = (double)((const T *)d.mass)[i];
        ke = 0.5 * m * d.mass_conv * ((double)v[0] * (double)v[0] + (double)v[1] * (double)v[1] + (double)v[2] * (double)v[2]);
    }
    seg_store(d, s, valid, ke);
}

/* ------------------------------------------------------------------ FIRE (O6) */
__device__ __forceinline__ void atomic_max_pos(double *dst, double v)
{
    atomicMax((unsigned long long *)dst, (unsigned long long)__double_as_longlong(v));
}

/* Fresh systems: v = 0, dt_start, alpha_start, counters 0.  sys_active = fresh or running. */
template <typename T>
__global__ void k_fire_init(DevState d, ts_fire_params p)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    int s = d.sysidx[i];
    int stt = d.f_status[s];
    if (stt == TS_FIRE_FRESH) {
        T *v = (T *)d.vel + 3 * i;
        v[0] = 0; v[1] = 0; v[2] = 0;
    }
    if (i == d.sysoff[s]) {
        if (stt == TS_FIRE_FRESH) {
            d.f_dt[s] = p.dt_start; d.f_alpha[s] = p.alpha_start; d.f_npos[s] = 0; d.f_nsteps[s] = 0;
        }
        d.sys_active[s] = (stt == TS_FIRE_FRESH || stt == TS_FIRE_RUNNING) ? 1 : 0;
        double *a = d.f_acc + 4 * (size_t)s;
        a[0] = 0.0; a[1] = 0.0; a[2] = 0.0; a[3] = 0.0;
    }
}

/* max_i |F_i|^2 of the fresh systems (their 0-step convergence test) */
template <typename T>
__global__ void k_fire_fmax(DevState d)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    int s = d.sysidx[i];
    if (d.f_status[s] != TS_FIRE_FRESH) return;
    const T *f = (const T *)d.force + 3 * i;
    double f2 = (double)f[0] * (double)f[0] + (double)f[1] * (double)f[1] + (double)f[2] * (double)f[2];
    atomic_max_pos(&d.f_acc[4 * (size_t)s], f2);
}

__global__ void k_fire_check0(DevState d, ts_fire_params p)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= d.S) return;
    if (d.f_status[s] == TS_FIRE_FRESH) {
        double *a = d.f_acc + 4 * (size_t)s;
        bool conv = sqrt(a[0]) < p.f_max;
        d.f_status[s] = conv ? TS_FIRE_CONVERGED : TS_FIRE_RUNNING;
        d.sys_active[s] = conv ? 0 : 1;
        a[0] = 0.0;
    }
}

/* (1) first half of the velocity-Verlet step with the system's own dt; max_steps check */
template <typename T>
__global__ void k_fire_pre(DevState d, ts_fire_params p)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    int s = d.sysidx[i];
    if (!d.sys_active[s]) return;
    bool failed = d.f_nsteps[s] >= p.max_steps;
    if (failed) {
        if (i == d.sysoff[s]) { d.f_status[s] = TS_FIRE_FAILED; d.sys_active[s] = 0; }
        return;
    }
    T *x = (T *)d.pos + 3 * i, *v = (T *)d.vel + 3 * i;
    const T *f = (const T *)d.force + 3 * i;
    T im = (T)1 / (((const T *)d.mass)[i] * (T)d.mass_conv);
    T dt = (T)d.f_dt[s], hdt = (T)0.5 * dt;
    T xx[3], vv[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        vv[k] = v[k] + hdt * (f[k] * im);
        xx[k] = x[k] + dt * vv[k];
        v[k] = vv[k]; x[k] = xx[k];
    }
    publish_pos<T>(d, i, s, xx[0], xx[1], xx[2]);
}

/* second half kick + the four per-system reductions: max|F|^2, P = F.v, v.v, F.F */
template <typename T>
__global__ void k_fire_post1(DevState d)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    bool valid = i < d.N;
    int s = valid ? d.sysidx[i] : 0;
    bool act = valid && d.sys_active[s];
    double f2 = 0, P = 0, vv = 0;
    if (act) {
        T *v = (T *)d.vel + 3 * i;
        const T *f = (const T *)d.force + 3 * i;
        T im = (T)1 / (((const T *)d.mass)[i] * (T)d.mass_conv);
        T hdt = (T)0.5 * (T)d.f_dt[s];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            T vk = v[k] + hdt * (f[k] * im);
            v[k] = vk;
            f2 += (double)f[k] * (double)f[k];
            P += (double)f[k] * (double)vk;
            vv += (double)vk * (double)vk;
        }
        atomic_max_pos(&d.f_acc[4 * (size_t)s], f2);
    }
    /* f_acc is [S,4]: max |F_i|^2 (an atomic max is order-independent), then the three sums in fixed order */
    const double part[3] = { P, vv, f2 };
    ts_sys_store<3, 1>(d, act ? s : -1, part);                   /* k_sum_fire adds the slots of every system */
}

/* P, v.v, F.F of the active systems from the partials of k_fire_post1: one warp per system, slot order */
__global__ void k_sum_fire(DevState d)
{
    const int s = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5);
    if (s >= d.S || !d.sys_active[s]) return;
    double tot[3];
    ts_sys_total<3>(d, s, 1, tot);
    if ((threadIdx.x & 31) == 0) {
        double *a = d.f_acc + 4 * (size_t)s;
        a[1] = tot[0]; a[2] = tot[1]; a[3] = tot[2];
    }
}

/* (2)..(5) per atom: freeze if converged, else mix (P > 0, with the alpha before its update) or
 * stop (P <= 0) */
template <typename T>
__global__ void k_fire_post2(DevState d, ts_fire_params p)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    int s = d.sysidx[i];
    if (!d.sys_active[s]) return;
    const double *a = d.f_acc + 4 * (size_t)s;
    if (sqrt(a[0]) < p.f_max) return;
    T *v = (T *)d.vel + 3 * i;
    if (a[1] > 0.0) {
        double fn = sqrt(a[3]), vn = sqrt(a[2]), al = d.f_alpha[s];
        if (fn > 0.0) {
            const T *f = (const T *)d.force + 3 * i;
            T cf = (T)(al * (vn / fn)), om = (T)(1.0 - al);
#pragma unroll
            for (int k = 0; k < 3; ++k) v[k] = om * v[k] + cf * f[k];
        }
    } else {
        v[0] = 0; v[1] = 0; v[2] = 0;
    }
}

__global__ void k_fire_sys(DevState d, ts_fire_params p)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= d.S) return;
    if (!d.sys_active[s]) return;
    double *a = d.f_acc + 4 * (size_t)s;
    d.f_nsteps[s] += 1;
    if (sqrt(a[0]) < p.f_max) {
        d.f_status[s] = TS_FIRE_CONVERGED;
        d.sys_active[s] = 0;
    } else if (a[1] > 0.0) {
        int np = d.f_npos[s] + 1;
        d.f_npos[s] = np;
        if (np > p.n_min) {
            double nd = d.f_dt[s] * p.f_inc;
            d.f_dt[s] = nd < p.dt_max ? nd : p.dt_max;
            d.f_alpha[s] = d.f_alpha[s] * p.f_alpha;
        }
    } else {
        d.f_dt[s] = d.f_dt[s] * p.f_dec;
        d.f_alpha[s] = p.alpha_start;
        d.f_npos[s] = 0;
    }
    a[0] = 0.0; a[1] = 0.0; a[2] = 0.0; a[3] = 0.0;
    d.sys_step[s] += 1ull;
}

/* ------------------------------------------------------------------ in-flight swap (a10) */
/* block k copies fresh system k into slot scratch[k]; scratch[n + k] = first fresh atom of k */
template <typename T>
__global__ void k_swap(DevState d, int n, const T *fpos, const T *fvel, const T *fmass,
                       const int *ftype, const T *fcell, const unsigned *fuid)
{
    int k = blockIdx.x;
    int slot = d.scratch[k];
    int src = d.scratch[n + k];
    int a0 = d.sysoff[slot], cnt = d.sysoff[slot + 1] - a0;
    T *pos = (T *)d.pos, *vel = (T *)d.vel, *mass = (T *)d.mass;
    int *type = (int *)d.type;
    for (int t = threadIdx.x; t < 3 * cnt; t += blockDim.x) {
        pos[3 * (size_t)a0 + t] = fpos[3 * (size_t)src + t];
        vel[3 * (size_t)a0 + t] = fvel ? fvel[3 * (size_t)src + t] : (T)0;
    }
    for (int t = threadIdx.x; t < cnt; t += blockDim.x) {
        if (fmass) mass[a0 + t] = fmass[src + t];
        if (ftype) type[a0 + t] = ftype[src + t];
    }
    if (threadIdx.x < 9 && fcell) ((T *)d.cell)[9 * (size_t)slot + threadIdx.x] = fcell[9 * (size_t)k + threadIdx.x];
    if (threadIdx.x == 0) {
        if (fuid) d.uid_own[slot] = fuid[k];
        d.f_status[slot] = TS_FIRE_FRESH;
        d.f_nsteps[slot] = 0;
        d.sys_step[slot] = 0ull;
        d.sys_active[slot] = 1;
        d.res_saved[slot] = 0;                  /* the resident engine's saved list belonged to the system that left */
    }
}

__global__ void k_fire_count(DevState d, int *out /* [2] converged, failed */)
{
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= d.S) return;
    int st = d.f_status[s];
    if (st == TS_FIRE_CONVERGED) atomicAdd(&out[0], 1);
    if (st == TS_FIRE_FAILED) atomicAdd(&out[1], 1);
}

/* kinetic energies of the systems this engine steps, from the partials of k_md_post / k_kinetic: one warp per system */
__global__ void k_sum_kinetic(DevState d)
{
    const int s = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5);
    if (s >= d.S || ts_skip(d, s)) return;
    double tot[1];
    ts_sys_total<1>(d, s, 1, tot);
    if ((threadIdx.x & 31) == 0) d.kinetic[s] = tot[0];
}

/* ------------------------------------------------------------------ host launchers */
#define ATOM_GRID(d) (unsigned)(((d).N + 255) / 256), 256
#define SYS_GRID(d) (unsigned)(((d).S + 127) / 128), 128
#define SYS_WARP_GRID(d) (unsigned)(((d).S + 3) / 4), 128      /* one warp per system */
#define BY_DTYPE(st, KERNEL, GRID, ...)                                              \
    do {                                                                             \
        if ((st)->d.dtype == TS_F32) KERNEL<float><<<GRID, 0, q>>>(__VA_ARGS__);     \
        else KERNEL<double><<<GRID, 0, q>>>(__VA_ARGS__);                            \
        (st)->launches += 1;                                                         \
    } while (0)

void launch_import(ts_state *st, cudaStream_t q) { BY_DTYPE(st, k_import, ATOM_GRID(st->d), st->d); }
void launch_md_pre(ts_state *st, const MdConst &c, cudaStream_t q) { BY_DTYPE(st, k_md_pre, ATOM_GRID(st->d), st->d, c); }
void launch_md_post(ts_state *st, const MdConst &c, bool want_ke, cudaStream_t q)
{
    BY_DTYPE(st, k_md_post, ATOM_GRID(st->d), st->d, c, want_ke ? 1 : 0);
    if (want_ke) { k_sum_kinetic<<<SYS_WARP_GRID(st->d), 0, q>>>(st->d); st->launches += 1; }
}
void launch_kinetic(ts_state *st, cudaStream_t q)
{
    BY_DTYPE(st, k_kinetic, ATOM_GRID(st->d), st->d);
    k_sum_kinetic<<<SYS_WARP_GRID(st->d), 0, q>>>(st->d);
    st->launches += 1;
}
void launch_fire_init(ts_state *st, const ts_fire_params &p, cudaStream_t q) { BY_DTYPE(st, k_fire_init, ATOM_GRID(st->d), st->d, p); }
void launch_fire_check0(ts_state *st, const ts_fire_params &p, cudaStream_t q)
{
    BY_DTYPE(st, k_fire_fmax, ATOM_GRID(st->d), st->d);
    k_fire_check0<<<SYS_GRID(st->d), 0, q>>>(st->d, p);
    st->launches += 1;
}
void launch_fire_pre(ts_state *st, const ts_fire_params &p, cudaStream_t q) { BY_DTYPE(st, k_fire_pre, ATOM_GRID(st->d), st->d, p); }
void launch_fire_post(ts_state *st, const ts_fire_params &p, cudaStream_t q)
{
    BY_DTYPE(st, k_fire_post1, ATOM_GRID(st->d), st->d);
    k_sum_fire<<<SYS_WARP_GRID(st->d), 0, q>>>(st->d);
    st->launches += 1;
    BY_DTYPE(st, k_fire_post2, ATOM_GRID(st->d), st->d, p);
    k_fire_sys<<<SYS_GRID(st->d), 0, q>>>(st->d, p);
    st->launches += 1;
}
void launch_fire_count(ts_state *st, cudaStream_t q)
{
    int *out = st->d.scratch + 2 * (size_t)st->d.S + 2;
    cudaMemsetAsync(out, 0, 2 * sizeof(int), q);
    k_fire_count<<<SYS_GRID(st->d), 0, q>>>(st->d, out);
    st->launches += 1;
}
void launch_swap(ts_state *st, int n, const ts_state_desc *fr, cudaStream_t q)
{
    if (st->d.dtype == TS_F32)
        k_swap<float><<<n, 256, 0, q>>>(st->d, n, (const float *)fr->pos, (const float *)fr->vel, (const float *)fr->mass,
                                       fr->type, (const float *)fr->cell, fr->sys_uid);
    else
        k_swap<double><<<n, 256, 0, q>>>(st->d, n, (const double *)fr->pos, (const double *)fr->vel, (const double *)fr->mass,
                                        fr->type, (const double *)fr->cell, fr->sys_uid);
    st->launches += 1;
}
