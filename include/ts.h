/*
 * ts.h -- C ABI of libts: batched pair-potential MD / FIRE on one B200 (sm_100a).
 *
 * The boundary named by BASELINE.json:north_star ("ts_state_create, ts_build_neighbors,
 * ts_compute_forces, ts_md_step, ts_fire_step") and laid out in SURVEY.md section 8(b).  The
 * operation is the paper's batched simulation: "The attributes of individual systems, such as
 * positions and momenta, are concatenated into a single SimState object ... concatenates atom-wise
 * ... and stacks batch-wise attributes (unit cell, stress tensor, etc.)" (section 3),
 * a model call that returns "energies, forces, and stress" (section 2) for the
 * classical potentials "Lennard-Jones, Morse, soft-sphere" (Abstract), advanced by
 * "molecular dynamics integrators" / "structural relaxation optimizers", with the
 * convergence check and swap of the InFlightAutobatcher (section 3).  The paper prints
 * no formula; the formulas are O1..O6 of SURVEY.md section 8(c), restated in DESIGN.md.
 *
 * Conventions
 *  - Plain C types only.  "device" = pointer into CUDA device memory of the current device,
 *    "host" = ordinary host memory.  `stream` is a cudaStream_t passed as void* (NULL = default).
 *  - Ownership: the CALLER owns every device array in ts_state_desc and the workspace blob; the
 *    library borrows them until ts_state_destroy and allocates no device memory itself.  The
 *    library owns only the host-side ts_state.  Outputs are written in place.
 *  - Layout at the boundary: [N,3] row-major positions / velocities / forces, [N] per-atom scalars,
 *    [S,3,3] cells whose ROWS are lattice vectors (x = f . h, all three directions periodic),
 *    per-atom system_idx non-decreasing 0..S-1.  All floating arrays of one state share `dtype`
 *    except energy / virial / kinetic, which are always float64.
 *  - Stored positions are never wrapped by the library.
 *  - Calls are asynchronous on `stream` unless stated.  A ts_state is not thread-safe.
 *  - Errors: argument errors return immediately (nothing enqueued).  Conditions found on the device
 *    (neighbour capacity overflow, image shift out of range, non-finite force, bad cell) set sticky
 *    bits in a device status word; ts_poll reports them, and once ts_poll has observed them every later
 *    stepping call returns TS_ERR_STICKY until ts_clear_error.  On overflow nothing is written past capacity.
 *  - Synchronising calls: ts_workspace_bytes, ts_state_create, ts_poll, ts_converged_mask, ts_swap_systems,
 *    ts_repack_systems, ts_get_neighbors, ts_set/get_system_steps, ts_clear_error; the first stepping call of the
 *    resident engine after create or after a swap / repack with new cells reads the cell geometry back once.
 *  - No CPU fallback exists: every entry point needs a CUDA device.
 */
#ifndef TS_H
#define TS_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ts_state ts_state;   /* opaque, host-side, owned by the library */
typedef int32_t ts_status;

enum {
    TS_OK = 0,
    TS_ERR_INVALID_ARG = 1,
    TS_ERR_CUDA = 2,
    TS_ERR_WORKSPACE_TOO_SMALL = 3,
    TS_ERR_NBR_OVERFLOW = 4,
    TS_ERR_STALE_NBR = 5,
    TS_ERR_NONFINITE = 6,
    TS_ERR_UNSUPPORTED = 7,
    TS_ERR_STICKY = 8
};

/* bits of ts_report.flags (device status word) */
enum {
    TS_FLAG_NBR_OVERFLOW = 1u,   /* neighbour list larger than the workspace capacity             */
    TS_FLAG_SHIFT_RANGE = 2u,    /* an image shift left [-16,15] (atom > 15 cells from its image)  */
    TS_FLAG_NONFINITE = 4u,      /* a non-finite force was produced                                */
    TS_FLAG_BAD_CELL = 8u        /* singular cell, or a stencil wider than 31 bins                 */
};

typedef enum { TS_F32 = 0, TS_F64 = 1 } ts_dtype;
typedef enum { TS_LJ = 0, TS_MORSE = 1, TS_SOFT_SPHERE = 2 } ts_pot_kind;
enum { TS_WANT_ENERGY = 1u, TS_WANT_VIRIAL = 2u };
enum { TS_NVE = 0, TS_BAOAB = 1 };
enum { TS_FIRE_FRESH = 0, TS_FIRE_RUNNING = 1, TS_FIRE_CONVERGED = 2, TS_FIRE_FAILED = 3 };

/* Units: a = F / (m * mass_conv).  metal: mass_conv = 103.64269652680505
 * (eV fs^2 / (amu A^2)), kB = 8.617333262145179e-5 eV/K; reduced units: 1, 1.                     */
typedef struct { double mass_conv; double kB; } ts_units;

/* Pair potential.  HOST tables [n_types*n_types], entry (ti*n_types + tj); copied at
 * create.  LJ:    V = 4 p0 [(p1/r)^12 - (p1/r)^6]                      p0 = eps, p1 = sigma
 * Morse:          V = p0 [(1 - exp(-p1 (r - p2)))^2 - 1]               p0 = D, p1 = alpha, p2 = r0
 * soft sphere:    V = (p0/p2) (1 - r/p1)^p2 for r < p1, else 0         p0 = eps, p1 = sigma, p2 = exponent
 * Pairs with r >= rc contribute exactly 0 (strict r^2 < rc^2).  shift_energy: V <- V - V(rc).     */
typedef struct {
    int32_t kind;            /* ts_pot_kind */
    int32_t n_types;
    const double *p0, *p1, *p2, *rc;
    int32_t shift_energy;
} ts_potential;

/* The batch.  All pointers device unless NULL is allowed.                           */
typedef struct {
    int64_t n_atoms;         /* N >= 1 */
    int32_t n_systems;       /* S >= 1 */
    int32_t dtype;           /* ts_dtype of pos, vel, force, mass, cell */
    ts_units units;
    void *pos;               /* [N,3] in/out */
    void *vel;               /* [N,3] in/out */
    void *force;             /* [N,3] out    */
    const void *mass;        /* [N]   in     */
    const int32_t *type;     /* [N]   in, 0..n_types-1 */
    const int32_t *system_idx; /* [N] in, non-decreasing; every system has >= 1 and <= 131072 atoms */
    const void *cell;        /* [S,3,3] in, rows = lattice vectors */
    double *energy;          /* [S]     out, potential energy E_s (float64) */
    double *virial;          /* [S,3,3] out, W_s = -dE/dstrain (float64); stress = -W/V */
    double *kinetic;         /* [S]     out, KE_s = 1/2 sum m mass_conv v^2 (float64) */
    const uint32_t *sys_uid; /* [S] persistent ids for the Philox counter (R18); NULL -> 0..S-1 */
} ts_state_desc;

/* skin: Verlet skin (list radius = max rc + skin; rebuild when an atom moved > skin/2).
 * slack: capacity factor on the estimated pair count (>= 1; 0 -> 1.25).                           */
typedef struct { double skin; double slack; } ts_nbr_params;

/* integrator TS_NVE: velocity Verlet.  TS_BAOAB: Langevin B A O A B (O4) with one
 * Philox4x32-10 block per atom per step, key = seed, counter = (local atom index, sys_uid,
 * step lo, step hi) (O5).  friction in 1/time, temperature in K (uses units.kB).                  */
typedef struct { int32_t integrator; double dt, temperature, friction; uint64_t seed; } ts_md_params;

/* FIRE, MD form: Bitzek et al., PRL 97, 170201 (2006).                                */
typedef struct {
    double dt_start, dt_max, f_inc, f_dec, alpha_start, f_alpha, f_max;
    int32_t n_min, max_steps;
} ts_fire_params;

typedef struct {
    uint32_t flags;          /* TS_FLAG_* sticky bits */
    int32_t n_rebuilds;      /* general engine: build events since create in which at least one system was rebuilt */
    int64_t nnz;             /* directed pairs in the current list (resident engine: summed over the systems' lists) */
    int64_t nnz_capacity;
    int64_t steps_done;      /* MD/FIRE steps enqueued since create */
    int32_t n_converged;     /* systems with FIRE status converged */
    int32_t n_failed;        /* systems that hit max_steps */
    int32_t max_neighbors;   /* longest row built since the last full build (general engine; a running maximum over per-system rebuilds) */
    int32_t list_valid;
    int64_t resident_rebuilds; /* per-system list builds since create, summed over systems (both engines) */
    int32_t engine;          /* engine that ran the last stepping call: 0 general, 1 resident, 2 both (mixed dispatch of a ragged batch) */
    int32_t reserved;
} ts_report;

/* Bytes of workspace ts_state_create needs for this batch (the memory-estimate primitive, SURVEY
 * a9).  Reads the cells from the device (synchronises).                                           */
ts_status ts_workspace_bytes(const ts_state_desc *desc, const ts_potential *pot,
                             const ts_nbr_params *nbr, size_t *out_bytes);

/* Host-only variant of the same estimate for one system of n_atoms in volume `volume`: bytes of
 * workspace plus boundary arrays that system adds to a batch.  No device needed.                  */
ts_status ts_estimate_system_bytes(int64_t n_atoms, double volume, double r_list, double slack,
                                   int32_t dtype, size_t *out_bytes);

/* Create a state over caller-owned arrays.  workspace: device, 256-byte aligned, workspace_bytes >=
 * ts_workspace_bytes.  Validates system_idx (synchronises once).  Imports pos/vel.               */
ts_status ts_state_create(const ts_state_desc *desc, const ts_potential *pot,
                          const ts_nbr_params *nbr, void *workspace, size_t workspace_bytes,
                          ts_state **out);
ts_status ts_state_destroy(ts_state *st);

/* Cell-list neighbour build from the current desc.pos: binning + counting sort by
 * (system, cell), then ONE search pass that buffers each row, reserves its place in the system's CSR
 * segment with one atomic and copies it out (rows of any length; capacity check per system: on
 * overflow nothing is written past the segment, TS_FLAG_NBR_OVERFLOW is set and the list is invalid). */
ts_status ts_build_neighbors(ts_state *st, void *stream);

/* Forces (always), energy / virial when asked from the current desc.pos; rebuilds
 * the list first if it is missing or an atom moved more than skin/2 since the last build.        */
ts_status ts_compute_forces(ts_state *st, uint32_t want, void *stream);

/* n_steps of MD entirely on the device, skin checks and rebuilds included.  On
 * return of the enqueued work: pos, vel at t + n dt, force = F(pos), energy, kinetic (and virial if
 * want has TS_WANT_VIRIAL) of the final state (R16).                                              */
ts_status ts_md_step(ts_state *st, const ts_md_params *p, int32_t n_steps, uint32_t want,
                     void *stream);

/* Up to n_steps of FIRE on every system that is not frozen.  Fresh systems are
 * initialised (v = 0, dt_start, alpha_start) and checked for convergence with 0 steps.  Converged
 * and failed systems are left bit-unchanged.                                                      */
ts_status ts_fire_step(ts_state *st, const ts_fire_params *p, int32_t n_steps, void *stream);

/* Synchronises `stream` and reports.  Returns TS_OK even when flags are set (read out->flags).    */
ts_status ts_poll(ts_state *st, ts_report *out, void *stream);

/* Synchronising read of the per-system FIRE status into HOST arrays (any may be NULL):
 * mask[s] = 1 when converged; status[s] = TS_FIRE_*; fire_steps[s] = steps taken so far.          */
ts_status ts_converged_mask(ts_state *st, uint8_t *mask, int32_t *status, int32_t *fire_steps,
                            void *stream);

/* (InFlightAutobatcher: "after every few steps ... convergence function" -- the check must not stall the device.)
 * The same status words WITHOUT synchronising: status[s] and fire_steps[s] (HOST arrays of S int32, either may be
 * NULL) are filled by copies enqueued on `stream` behind the work already there; they are valid once the caller has
 * waited for that point of the stream (an event recorded after this call).  The arrays should be page-locked
 * (cudaHostAlloc / a pinned torch tensor): with pageable memory CUDA falls back to a copy that blocks the host.
 * Lets an in-flight scheduler enqueue the next ts_fire_step before it has read the result of the last one: systems
 * that converged meanwhile stay bit-unchanged (R22), so acting on a status that is one call old changes no result. */
ts_status ts_fire_status_async(ts_state *st, int32_t *status, int32_t *fire_steps, void *stream);

/* In-flight swap, equal sizes (ts_repack_systems: any sizes).  Synchronises `stream`; the
 * stepping call that follows a swap with new cells re-plans the resident engine (one small device read).
 * Replaces the systems in `slots` (HOST, n entries) by the
 * n systems of `fresh` (device arrays pos, vel, mass, type, cell, sys_uid; system k of fresh must
 * have exactly as many atoms as slot slots[k]).  Their FIRE state becomes fresh, their step
 * counter 0, and the neighbour list is marked stale.                                              */
ts_status ts_swap_systems(ts_state *st, const int32_t *slots, int32_t n, const ts_state_desc *fresh,
                          void *stream);

/* Ragged in-flight replacement (Fig. 3): the batch becomes the systems
 * keep[0..n_keep) of the current batch (HOST slot numbers, each at most once, in the order given) followed by the
 * systems of `fresh` (device arrays pos, vel (NULL: zero), mass, type, cell, sys_uid (NULL: slot number);
 * fresh_n_atoms HOST [fresh->n_systems]; NULL fresh: compaction only), of any sizes.  Kept systems keep positions,
 * velocities, FIRE state, step counters and uids; fresh ones start FRESH at step 0.  n_atoms, n_systems and the
 * neighbour list are re-laid; energy / virial / kinetic of a slot are stale until the next force evaluation.  The new
 * batch must fit what the state was created with (ts_get_capacity: atoms, systems, pair slots), else
 * TS_ERR_WORKSPACE_TOO_SMALL and nothing has changed.  Synchronises `stream`.                                      */
ts_status ts_repack_systems(ts_state *st, const int32_t *keep, int32_t n_keep, const ts_state_desc *fresh,
                            const int32_t *fresh_n_atoms, void *stream);

/* Capacity of a state (sizes at create) and the pair slots one system needs (the paper's n_atoms x density scaler,
 * PAPER.md:88, with the coefficient the library uses): what an admission rule has to add up before a repack.       */
ts_status ts_get_capacity(const ts_state *st, int64_t *n_atoms, int32_t *n_systems, int64_t *n_pairs);
ts_status ts_estimate_system_pairs(int64_t n_atoms, double volume, double r_list, double slack, int64_t *out_pairs);

/* Synchronising export of the current list to HOST arrays (test / graph export): off [N+1], and
 * for each directed pair its GLOBAL neighbour index j and image shift S (relative to the stored
 * positions, R6).  cap = capacity of j / shift in pairs; TS_ERR_WORKSPACE_TOO_SMALL if nnz > cap. */
ts_status ts_get_neighbors(ts_state *st, int64_t *off, int32_t *j, int8_t *shift, int64_t cap,
                           void *stream);

/* The Verlet list the system-resident engine would step system `system` with at the current positions, decoded to
 * HOST arrays like ts_get_neighbors (off [n_s + 1] relative to the system, GLOBAL j, shift relative to the stored
 * positions).  It is a SUPERSET list: every pair within max rc + skin is in it, and nothing beyond that radius plus a
 * few parts in 10^6 of the longest cell edge (fixed-point fractions); the pair loop applies the strict cutoff (R9).
 * j / shift may be NULL to get the count (*nnz) only.  TS_ERR_UNSUPPORTED when the resident engine does not apply to
 * the batch.  Uses the pair region of the workspace (the general engine's list is invalidated).  Synchronises.       */
ts_status ts_get_resident_neighbors(ts_state *st, int32_t system, int64_t *off, int32_t *j, int8_t *shift,
                                    int64_t cap, int64_t *nnz, void *stream);

/* ---- graph export and external-model stepping (SURVEY 8(f) NEXT-2; PAPER.md:56 ModelInterface, :112) ------------
 * The current Verlet list (radius max rc + skin, general engine; built or skin-checked first) as a dense edge list in
 * DEVICE arrays: edge_i / edge_j [cap] global atom indices, edge_shift [cap,3] in the state dtype = the integer image
 * shift S of the pair: r_ij = x_j - x_i + S . h with the STORED positions (R6).  *n_edges (device) = edges of the
 * list; when it exceeds cap only the first cap edges are written.  Edges of a system are contiguous, systems in batch
 * order.  Asynchronous on `stream`.                                                                                 */
ts_status ts_export_edges(ts_state *st, int64_t *edge_i, int64_t *edge_j, void *edge_shift, int64_t cap,
                          int64_t *n_edges, void *stream);

/* (Same operation as ts_export_edges: PAPER.md:56 ModelInterface, :112 graph construction.)
 * ts_export_edges for callers that must not allocate and cannot lend workspace scratch (code under CUDA graph
 * capture, tight serving loops): same arguments, same result, but the per-system exclusive scan of the edge counts
 * lives in a file-scope device array of the library instead of a workspace region.  No cudaMalloc / cudaFree or
 * allocating library routine is called (no entry point of this library allocates device memory; this one also
 * borrows none from the workspace for its scratch).
 *   limit      at most 16,384 systems in the state (the array holds 16,385 int64 = 131,080 bytes on every GPU that
 *              loads the library, until the process exits); more: TS_ERR_WORKSPACE_TOO_SMALL, ts_last_error names
 *              the limit, nothing is launched, use ts_export_edges.
 *   sharing    ONE array per GPU, shared by every state and every call; it keeps the contents of the last call.  Each
 *              call rewrites the entries it reads before reading them, so nothing needs clearing -- but two calls that
 *              overlap on the GPU (different streams, no ordering between them) race on it and give wrong edges.
 *   set-up     the device address of the array is looked up once per device on the first call with that device
 *              current; ts_static_scratch_setup does the same ahead of time (call it before a stream capture starts).
 * ts_static_scratch_setup: *max_systems (host, may be NULL) = the limit; TS_ERR_CUDA if the lookup fails.            */
ts_status ts_export_edges_static(ts_state *st, int64_t *edge_i, int64_t *edge_j, void *edge_shift, int64_t cap,
                                 int64_t *n_edges, void *stream);
ts_status ts_static_scratch_setup(int64_t *max_systems);

/* One MD / FIRE step split around a force evaluation the CALLER enqueues on `stream` (an external energies / forces /
 * stress provider writing desc.force, and desc.energy / desc.virial if it wants them reported):
 *   MD:   TS_PHASE_INIT (list for the current positions) -> caller: F(x) -> then per step
 *         TS_PHASE_PRE (B A (O A), skin check, rebuild if due: ts_export_edges is current) -> caller: F(x) ->
 *         TS_PHASE_POST (B, kinetic energy, step counters += 1).
 *   FIRE: TS_PHASE_INIT (fresh systems: v = 0, dt_start, alpha_start; list) -> caller: F(x) -> TS_PHASE_CHECK0 (the
 *         0-step convergence test) -> per step TS_PHASE_PRE -> caller: F(x) -> TS_PHASE_POST (second half kick,
 *         reductions, FIRE state machine; frozen systems stay bit-unchanged).
 * Same integrator kernels as ts_md_step / ts_fire_step of the general engine.  Asynchronous.                         */
enum { TS_PHASE_INIT = 0, TS_PHASE_PRE = 1, TS_PHASE_POST = 2, TS_PHASE_CHECK0 = 3 };
ts_status ts_md_step_external(ts_state *st, const ts_md_params *p, int32_t phase, void *stream);
ts_status ts_fire_step_external(ts_state *st, const ts_fire_params *p, int32_t phase, void *stream);

/* Per-system step counters used by the Philox counter (R18): HOST [S] in / out.  Synchronising.   */
ts_status ts_set_system_steps(ts_state *st, const uint64_t *steps, void *stream);
ts_status ts_get_system_steps(ts_state *st, uint64_t *steps, void *stream);

/* Select the stepping engine: 0 = general multi-kernel path (any system size), 1 = system-resident
 * path (whole systems held in shared memory across steps) for every system it can hold (cell heights >= 2 r_list,
 * <= 2048 atoms), in up to four size classes launched side by side; ts_md_step steps the other systems of a ragged
 * batch with the general engine NEXT to it on a stream of its own (ts_fire_step: all systems or none).  Default 1.
 * Results obey the same tolerances either way.                                                                     */
ts_status ts_set_engine(ts_state *st, int32_t engine);

/* Tell the library that the caller wrote desc.pos / desc.vel from outside (e.g. a host -> device
 * copy): forces are stale and the list must be skin-checked against the new positions before the
 * next step (the system-resident engine, which keeps its lists from one call to the next in the
 * pair region of the workspace, builds them anew).  REQUIRED after such a write: without it the
 * resident engine would go on with lists made for the old positions.  Host-side flag only,
 * enqueues nothing.                                                                               */
ts_status ts_invalidate(ts_state *st);

/* Register-only FMA microbenchmark: the ALU peak the roofline of the pair kernels is reported against.
 * kind 0: fp32 FFMA, 1: fp64 DFMA, 2: packed fp32 (fma.rn.f32x2).  scratch: device, >= 4096 bytes.  Synchronises.   */
ts_status ts_measure_fma_tflops(int32_t kind, void *scratch, double *tflops, void *stream);

/* Number of kernel launches enqueued by this state since create (for bench accounting).           */
int64_t ts_launch_count(const ts_state *st);

/* ---- host-side scheduling primitives (no device needed; all arrays HOST) ------------------------
 * cost / scaler values are in any one unit (bytes from ts_estimate_system_bytes, or the paper's
 * n_atoms / n_atoms_x_density memory scaler).                                        */

/* In-flight admission: the longest prefix of cost[0..n) whose sum stays <= budget.  */
ts_status ts_sched_fill(const double *cost, int64_t n, double budget, int64_t *n_taken, double *used);

/* Figure 2 step 4: min over probes of n_systems[k] * scaler[k].                  */
ts_status ts_sched_max_scaler(const int64_t *n_systems, const double *scaler, int32_t n_probes, double *out);

/* BinningAutobatcher: first-fit-decreasing 1-D bin packing; bin_of[k] = bin of system
 * k, *n_bins = bins used.  TS_ERR_INVALID_ARG if a system exceeds the capacity.                   */
ts_status ts_sched_binpack(const double *cost, int64_t n, double capacity, int32_t *bin_of, int32_t *n_bins);

/* Multi-GPU sharding by system (no exchange step): longest-processing-time-first
 * assignment; rank_of[k] = rank of system k, load[r] = summed cost of rank r (may be NULL).        */
ts_status ts_sched_partition(const double *cost, int64_t n, int32_t n_ranks, int32_t *rank_of, double *load);

ts_status ts_clear_error(ts_state *st, void *stream);
const char *ts_status_string(ts_status s);
const char *ts_last_error(const ts_state *st);

#ifdef __cplusplus
}
#endif
#endif /* TS_H */
