/* emx.h -- C-ABI boundary of the B200-native EM-shower step loop.
 *
 * The hot path of arxiv 2203.09467 ("Celeritas"): the per-track Monte Carlo step
 * loop of a coupled gamma / e- / e+ electromagnetic shower.  The calls follow the
 * paper's statement of the problem -- inputs are geometry, physics, events,
 * cutoff thresholds and scoring regions (scoring API
 * PAPER.md:152); the loop is PAPER.md:114 ("six characteristics")
 * (tabulated cross sections, per-model interaction kernels)
 * (secondary stack allocator), PAPER.md:204-212 (slots, queued initializers,
 * iteration until nothing is left), PAPER.md:142 (surfaces + CSG cells) and
 * PAPER.md:144 (field propagation).  The readings of everything the paper
 * leaves open are listed in DESIGN.md section 3.
 *
 * Conventions
 *   - plain C, no torch types.  Every pointer is marked HOST or DEVICE.
 *   - units: MeV, cm, g/cm3, tesla.  Particle codes 0 = gamma, 1 = e-, 2 = e+.
 *   - all floating point is IEEE fp64; integers are 32 bit unless stated.
 *   - every call returns 0 (or a non-negative id) on success and a negative
 *     EMX_E_* code on failure; emx_last_error() gives the text.  Nothing
 *     throws or aborts across the boundary.
 *   - bulk device memory (primaries, workspace = track store + queues +
 *     tallies) is allocated by the CALLER and passed as raw device pointers
 *     together with the CUDA stream handle (cudaStream_t as void*; NULL = the
 *     legacy default stream).  The library owns only the problem description
 *     and one small (< 1 MB) device block holding tables and geometry.
 *   - calls on one emx_problem are not thread-safe.
 *   - there is NO CPU fallback: without a CUDA device every compute call
 *     returns EMX_E_CUDA.
 */
#ifndef EMX_H
#define EMX_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EMX_MAX_ELEM 4   /* elements per material */
#define EMX_MAX_FACES 8  /* faces per cell */

/* error codes */
#define EMX_OK 0
#define EMX_E_ARG (-1)      /* invalid argument */
#define EMX_E_STATE (-2)    /* call out of order (e.g. tables not built) */
#define EMX_E_CUDA (-3)     /* CUDA runtime error or no device */
#define EMX_E_CAPACITY (-4) /* workspace too small / secondary stack cannot make progress */
#define EMX_E_NOMEM (-5)

/* surface types ("quadric surfaces", restricted): f = x_a - v (planes), x^2+y^2 - v^2 (CZ) */
#define EMX_S_PX 0
#define EMX_S_PY 1
#define EMX_S_PZ 2
#define EMX_S_CZ 3

/* process mask bits (Table 2) */
#define EMX_M_COMPTON 1u
#define EMX_M_PHOTO 2u
#define EMX_M_PAIR 4u
#define EMX_M_IONI 8u   /* Moller + Bhabha */
#define EMX_M_BREMS 16u
#define EMX_M_ANNIH 32u

/* process ids (interaction counters, step results) */
#define EMX_P_COMPTON 0
#define EMX_P_PHOTO 1
#define EMX_P_PAIR 2
#define EMX_P_MOLLER 3
#define EMX_P_BHABHA 4
#define EMX_P_BREMS 5
#define EMX_P_ANNIH 6
#define EMX_P_REST 7 /* e+ annihilation at rest */
#define EMX_NPROC 8

/* Steps-per-track histogram ("steps per track ... by particle type", one of the two observables
 * of the paper's verification problem).  A track that took n >= 1 steps falls into bin n below 16; above, every
 * octave has four equal bins: 16 + 4 (e - 4) + (the two bits of n below its leading bit), e = floor(log2 n);
 * the last bin collects everything beyond. */
#define EMX_NHIST 96

/* what limited the step */
#define EMX_A_NONE 0
#define EMX_A_DISCRETE 1
#define EMX_A_LOSS 2
#define EMX_A_BOUNDARY 3
#define EMX_A_TRUNC 4 /* vacuum step cap / field substeps exhausted */
#define EMX_A_MSC 5   /* multiple-scattering step limit (emx_physics.msc) */

/* table kinds per material, each n_E doubles on the log grid */
#define EMX_T_COMPTON 0
#define EMX_T_PHOTO 1
#define EMX_T_PAIR 2
#define EMX_T_MOLLER 3
#define EMX_T_BREMS_EM 4
#define EMX_T_DEDX_EM 5
#define EMX_T_RANGE_EM 6
#define EMX_T_BHABHA 7
#define EMX_T_BREMS_EP 8
#define EMX_T_ANNIH 9
#define EMX_T_DEDX_EP 10
#define EMX_T_RANGE_EP 11
#define EMX_T_PAIR_ELEM0 12 /* + element index: n_i * sigma_pair(Z_i) for element selection */
#define EMX_T_MSC (EMX_T_PAIR_ELEM0 + EMX_MAX_ELEM) /* 1 / lambda_1: inverse first transport mean free path of e+-, 1/cm */
#define EMX_T_VAR_EM (EMX_T_MSC + 1) /* d(variance of the restricted collision loss)/ds of e-, MeV2/cm */
#define EMX_T_VAR_EP (EMX_T_MSC + 2) /* ... of e+ */
#define EMX_T_MSC2 (EMX_T_MSC + 3) /* 1 / lambda_2: inverse second transport mean free path of e+- (msc = 2), 1/cm */
#define EMX_NTABLE (EMX_T_MSC + 4)

typedef struct emx_problem emx_problem; /* opaque, owned by the library */

/* physics switches and numerical parameters (PAPER.md:114 ii, iii, vi; PAPER.md:236 cutoffs).
 * emx_create() fills in the defaults quoted in DESIGN.md (R9, R14). */
typedef struct {
    uint32_t process_mask;      /* EMX_M_* */
    double E_min, E_max;        /* energy grid, MeV */
    int32_t n_E;                /* grid points, >= 2 */
    double E_trk;               /* tracking cut, MeV */
    double prod_cut_cm;         /* > 0: derive per-material production thresholds from this length */
    double alpha_R, rho_R;      /* continuous-loss step function (rho_R in cm) */
    double lin_loss;            /* linear-loss limit as a fraction of E */
    double field_eps;           /* cm: RK4 local error and boundary landing tolerance */
    int32_t max_substeps;       /* field substep attempts per step */
    double vacuum_step;         /* cm: step cap in vacuum */
    int32_t max_steps;          /* per track; then the track is killed into looper_lost */
    int32_t deposit_e_at_creation; /* 1: every e- is deposited where it is born (BASELINE configs[0]) */
    /* Multiple scattering of e+- (Table 2: "Multiple scattering: Urban, WentzelVI", in progress
     * there, no formula printed; DESIGN.md R-MSC).  msc = 1: 1/lambda_1 is tabulated from the screened-Rutherford
     * transport cross section (Moliere screening, nuclear-size cutoff); a step of e+- in matter is limited to
     * max(msc_fr * max(range, lambda_1), msc_smin) and ends with a deflection drawn from the Henyey-Greenstein
     * law of mean cosine exp(-s (1/lambda_1(E) + 1/lambda_1(E')) / 2) (two draws, taken right after draw 0).
     * msc = 2 (DESIGN.md R-MSC2) adds the spatial moments of Lewis' theory: 1/lambda_2 is tabulated too
     * (EMX_T_MSC2); the step limits are TRUE path lengths t and the track is moved by the mean geometric length
     * lambda_1 (1 - exp(-t / lambda_1)); after the deflection a step that did not end on a boundary is shifted
     * sideways, along the transverse part of the new direction, with the mean square <x^2 + y^2> of the theory,
     * at most 0.9 of the way to the cell's boundary.  emx_step_result.s and the energy loss refer to the true path. */
    int32_t msc;
    double msc_fr;              /* > 0 */
    double msc_smin;            /* cm, > 0 */
    /* Energy-loss fluctuations of e+- (PAPER.md:114 ii continuous slowing down; DESIGN.md R-FLUCT).  fluct = 1:
     * the variance of the collisions below the production threshold per unit path, n_e Int_0^Tup W^2 dsigma of the
     * Moller / Bhabha laws, is tabulated (EMX_T_VAR_*); the continuous loss of a step is drawn from the normal law
     * about its mean with that variance times s, clamped to [0, min(2 mean, E)] (two draws, taken right after
     * draw 0 and before those of the multiple scattering); a range stop is not fluctuated. */
    int32_t fluct;
    /* Integrator of the field propagation ("different integration algorithms"): 0 = classical RK4 with step
     * doubling (C9; what B:configs names), 1 = the embedded Dormand-Prince 5(4) pair (DESIGN.md R-INT) --
     * same step-size rule, boundary search and landing tolerance, fewer and longer substeps on smooth stretches. */
    int32_t integrator;
} emx_physics;

/* run totals (PAPER.md:176 energy deposition; Fig. 5 diagnostics PAPER.md:204-212) */
typedef struct {
    double escaped, below_cut, looper, E_in; /* MeV */
    uint64_t steps[3];                       /* track-steps by particle type */
    uint64_t tracks[3];                      /* tracks created by particle type (primaries included) */
    uint64_t inter[EMX_NPROC];               /* discrete interactions by process id */
    uint64_t null_int;                       /* kinematically impossible (null) interactions */
    uint64_t track_steps;                    /* sum of steps[] */
    uint64_t stalls;                         /* steps re-executed because the secondary stack was full */
    uint64_t iterations;                     /* step iterations of the loop */
    uint64_t peak_live, peak_queue;          /* max tracks in flight / queued initializers */
} emx_scalars;

/* one track, array-of-structures form used only by the level-2 parity hook emx_step_batch */
typedef struct {
    double x[3], u[3], E;
    uint64_t tid;
    uint32_t prim, step;
    int32_t vol, surf, ptype, alive;
} emx_track;

/* everything one step produces (emx_step_batch output) */
typedef struct {
    emx_track trk;          /* updated track, alive = 0 if killed */
    int32_t action;         /* EMX_A_* */
    int32_t process;        /* EMX_P_* or -1 */
    int32_t n_sec;
    emx_track sec[4];       /* allocated secondaries in ordinal order */
    int32_t sec_ord[4];
    double edep;            /* MeV deposited, belongs to cell edep_vol */
    int32_t edep_vol;
    double below_cut;       /* part of edep from tracking-cut kills / births */
    double escaped, looper;
    double s;               /* step length travelled, cm */
    double msc_tau;         /* path length / lambda_1 behind this step's multiple-scattering deflection (0: none) */
    int32_t n_draws;        /* uniforms consumed */
    int32_t null_int;
    int32_t rest;           /* e+ annihilated at rest in this step */
    int32_t n_sub;          /* substep attempts of the field propagation behind this step (0: straight move) */
} emx_step_result;

/* ---- problem description (host side; arrays are HOST pointers, copied during the call) ---- */

/* New problem with default physics.  *out receives the handle. */
int emx_create(emx_problem **out);
void emx_destroy(emx_problem *p);

/* Material (PAPER.md:114 i "material-dependent physical properties"): n_elem <= EMX_MAX_ELEM elements
 * with atomic number Z, molar mass A (g/mol) and mass fraction; density g/cm3; mean excitation energy in
 * eV (> 0).  Returns the material id (>= 0); vacuum is material -1 and is never added. */
int emx_add_material(emx_problem *p, int n_elem, const int *Z, const double *A, const double *mass_frac,
                     double density_g_cm3, double mean_exc_energy_eV);

/* Surface: type EMX_S_*, value = plane position or cylinder radius (cm).  Returns its id. */
int emx_add_surface(emx_problem *p, int type, double value_cm);

/* Cell = conjunction of n_faces <= EMX_MAX_FACES half-spaces (surface id, sense -1: f < 0 side, +1: f > 0
 * side); material id or -1 (vacuum); tally id or -1 (not scored).  Cells must tile the world without
 * overlap; leaving every cell = escape.  Returns the cell id. */
int emx_add_volume(emx_problem *p, int n_faces, const int *surf, const int *sense, int material, int tally);

/* Uniform magnetic field in tesla; all zero = no field. */
int emx_set_field(emx_problem *p, double Bx_T, double By_T, double Bz_T);

/* Non-uniform field ("propagation of particles through arbitrary magnetic fields"):
 * turns the field set with emx_set_field, which must point along +-z, into a solenoid field that falls off
 * towards the ends:  B(x) = |B| g(x),  f(z) = 1 / (1 + exp((|z| - z0) / a)),
 * g = (-x f'(z) / 2, -y f'(z) / 2, f(z)),  f' = -sign(z) f (1 - f) / a  (div B = 0 to first order in r).
 * The adaptive RK4 then takes the field at its stage positions.  z0, a in cm, both > 0; EMX_E_ARG otherwise or
 * when the field is not along z.  emx_set_field resets to a uniform field.  Invalidates the tables. */
int emx_set_field_fringe(emx_problem *p, double z0_cm, double a_cm);

int emx_get_physics(const emx_problem *p, emx_physics *out);
int emx_set_physics(emx_problem *p, const emx_physics *ph);

/* Explicit production thresholds (MeV) for one material instead of the cut-length conversion. */
int emx_set_cuts(emx_problem *p, int material, double Tcut_MeV, double kcut_MeV);

/* ---- tables (BASELINE configs[0] "tabulated from closed forms") ---- */

/* Runs the table-builder kernels on `stream`, uploads geometry, and synchronises the stream. */
int emx_build_tables(emx_problem *p, void *stream);

/* Copies one table (n == n_E doubles) of a material to HOST memory. */
int emx_get_table(const emx_problem *p, int material, int kind, double *host_out, int n);

/* host_out8 = { n_e [1/cm3], I [MeV], plasma energy [MeV], X0 [cm], Tcut [MeV], kcut [MeV], rho, n_elem } */
int emx_get_material_info(const emx_problem *p, int material, double *host_out8);

int emx_n_tally(const emx_problem *p);

/* ---- transport ---- */

/* Bytes of caller-provided DEVICE workspace for a track store of n_slots and secondary stacks holding
 * queue_capacity records in total.  0 on invalid arguments. */
size_t emx_workspace_bytes(const emx_problem *p, long n_slots, long queue_capacity);

/* Transport n_primaries primaries to completion.  ptype[n], E[n] (MeV), pos3[3n], dir3[3n] (unit vectors),
 * start_vol[n] (cell ids), start_surf[n] (surface the primary sits on or -1; may be NULL = all -1) are
 * DEVICE pointers in array-of-xyz layout; they are read, never written.  `workspace` is a DEVICE buffer of
 * at least emx_workspace_bytes() bytes, 256-byte aligned, owned by the caller; its contents are
 * overwritten.  Work is enqueued on `stream`; the call returns after the loop has finished and the run
 * totals are on the host (the loop itself is device-driven; the host waits once at the end).
 * Tallies accumulate in the problem's device block until emx_reset_tallies(). */
int emx_transport(emx_problem *p, long n_primaries, const int *ptype, const double *E, const double *pos3,
                  const double *dir3, const int *start_vol, const int *start_surf, uint64_t seed,
                  long n_slots, long queue_capacity, void *workspace, size_t workspace_bytes, void *stream);

/* Same call with every primary array in HOST memory (pageable or pinned): uploads on `stream`,
 * transports, and leaves the tallies readable.  This is the end-to-end entry bench.py times as `e2e`.
 * The primaries are staged in the caller's workspace: workspace_bytes must be at least
 * emx_workspace_bytes(n_slots, queue_capacity) + emx_staging_bytes(n_primaries) (EMX_E_CAPACITY otherwise); the
 * library allocates nothing. */
int emx_transport_host(emx_problem *p, long n_primaries, const int *ptype, const double *E,
                       const double *pos3, const double *dir3, const int *start_vol, const int *start_surf,
                       uint64_t seed, long n_slots, long queue_capacity, void *workspace,
                       size_t workspace_bytes, void *stream);

/* Bytes emx_transport_host needs behind the workspace proper to stage n_primaries primaries (52 bytes each,
 * every array 256-byte aligned). */
size_t emx_staging_bytes(long n_primaries);

int emx_reset_tallies(emx_problem *p, void *stream);

/* Sharding by primaries ("particle events are decomposed across MPI ranks"): the
 * primaries passed to the following emx_transport calls are the primaries first, first + 1, ... of a longer
 * list.  A history depends on the seed and on its primary index only, so the tallies and counters of the parts
 * of a list, transported anywhere in any order with their offsets, sum to those of the whole list.
 * Default 0.  first + n must stay below 2^32 (EMX_E_ARG otherwise, here or in emx_transport). */
int emx_set_primary_offset(emx_problem *p, long first);

/* Scheduling of the loop (track slots, queued initializers, time per step iteration).  Nothing
 * here changes what a step computes: histories are keyed by (seed, primary, track id, step), so the counters of a
 * run are the same under every schedule and its tallies are the same up to the order of their sums.
 *   loop_node      1 (default): the whole loop is one CUDA graph with a WHILE node; 0: graphs of 8 iterations
 *                  launched in batches with a look at the done flag in between (also the fallback when the driver
 *                  refuses conditional nodes).
 *   slice_min / slice_max / slice_above   time slicing of the field propagation: while more
 *                  than slice_above tracks are live (< 0: n_slots / 32), a propagation that has used slice_min
 *                  substep attempts in this iteration is parked for the next one as soon as its pool has no
 *                  unstarted track left, and after slice_max attempts in any case.  Defaults 2 / 16 / -1.
 *   mev_per_slot   primaries are admitted while the shower energy in flight (admitted - deposited - escaped) is below
 *                  mev_per_slot x n_slots: the energy in flight is what fills the slots and, beyond them, the queue
 *                  (PAPER.md:204-206).  <= 0: 20 MeV.
 *   admit_below    primaries are admitted (in waves of n_slots / 256, 256..4096) only while fewer records than this
 *                  wait on the stacks (the queue is the memory limit); <= 0: 2 n_slots.
 *   blocks_per_sm  persistent 128-thread blocks per SM of each step kernel, in the order k_a<gamma>,
 *                  k_a<charged>, k_a0, k_field, k_a2, k_b<gamma>, k_b<charged>; 0 = default (5, 4, 6, 6 -- 5 with a field map --,
 *                  5, 4, 4: what the kernels' registers allow).  Entry 7 holds two switches
 *                  for shared-memory staging of hot table slices: bit 0 = k_field copies the geometry's face table to
 *                  shared memory, bit 1 = k_a<gamma> copies the photon tables (3 per material) -- instead of reading
 *                  them through L1.  Both measured SLOWER on B200 (profiles/r2_staging.md) and kept for that comparison. */
typedef struct {
    int32_t loop_node;
    int32_t slice_min, slice_max;
    int64_t slice_above;
    int32_t blocks_per_sm[8];
    int64_t admit_below;
    int32_t mev_per_slot;
    int32_t reserved;
} emx_schedule;
int emx_get_schedule(const emx_problem *p, emx_schedule *out);
int emx_set_schedule(emx_problem *p, const emx_schedule *in);

/* edep_host[n_tally] (MeV per tally id) and the run totals, copied to HOST memory. */
int emx_read_tallies(const emx_problem *p, double *edep_host, emx_scalars *out);

/* hist_host[3 * EMX_NHIST] (HOST memory): tracks of the last transport by particle type (gamma, e-, e+) and by
 * the bin of the number of steps they took before they ended (absorbed, below the tracking cut, escaped,
 * looper).  Sums to scalars.tracks[] per type.  EMX_E_STATE before the first transport. */
int emx_read_step_hist(const emx_problem *p, uint64_t *hist_host);

/* Milliseconds the last emx_transport spent between its first launch and the end of the loop,
 * measured with CUDA events on the caller's stream; < 0 if none. */
double emx_last_transport_ms(const emx_problem *p);

/* Per-kernel timing of the loop.  Normally emx_transport runs the whole loop as ONE CUDA graph (a WHILE node
 * whose body is 8 iterations, the two pools' kernel chains as parallel branches, and a kernel that sets the node's
 * condition from the done flag) on internal streams ordered after `stream`.  on = 1: the kernels are launched
 * one by one on `stream` instead and every launch is bracketed by CUDA events on that stream; on = 2: launched
 * one by one without the events (what a profiler can list).  emx_get_profile: ms9[9] = milliseconds of the last
 * transport spent in { k_a<gamma>, k_a<charged> (no field), k_a0, k_field, k_a2 (field), k_b<gamma>,
 * k_b<charged>, refill (k_plan + k_fill + k_move), all step kernels }; *launches = kernels launched by the last
 * transport (always counted); *iterations_launched = iterations run, empty ones included (>= iterations needed:
 * the done flag is looked at once per 8 iterations in the graph, once per batch of launches otherwise).
 * emx_get_lanes: lanes8[0..6] = track slots processed by those seven kernels over the last transport (the units
 * of each kernel's algorithmic bytes), lanes8[7] = substep attempts of the field propagation.  Output pointers
 * may be NULL. */
int emx_set_profile(emx_problem *p, int on);
int emx_get_profile(const emx_problem *p, double *ms9, long *launches, long *iterations_launched);
int emx_get_lanes(const emx_problem *p, uint64_t *lanes8);

/* Per-iteration diagnostics of the last transport (Fig. 5): up to `max_iter` rows of
 * { live tracks, queued initializers } as uint32 pairs in HOST memory; returns rows written. */
long emx_get_iteration_log(const emx_problem *p, uint32_t *host_out, long max_iter);

/* Time per step iteration of the last transport (Fig. 5b), recorded when profiling is on:
 * up to `max_iter` rows of { refill ms, step-kernel ms } as float pairs in HOST memory; returns rows written
 * (iterations enqueued after the loop finished are included and cost only their launch overhead). */
long emx_get_iteration_times(const emx_problem *p, float *host_out, long max_iter);

/* ---- parity hooks ---- */

/* Level-2 parity hook: one step of each of n tracks with the same device step function the loop uses.
 * in[n] and out[n] are DEVICE pointers (AoS). */
int emx_step_batch(emx_problem *p, uint64_t seed, long n, const emx_track *in, emx_step_result *out,
                   void *stream);

/* Level-2 parity hook for ONE substep of the field propagation (C9): for each of n states
 * (x, u, curvature kappa [1/cm, signed], trial step h [cm]) one substep of the problem's integrator in the problem's
 * field, exactly as the propagation kernel runs it -- integrator 0: one RK4 step of h against two of h / 2, x1, u1 =
 * state after the two half steps, err = |x_full - x_half|; integrator 1: one Dormand-Prince step, x1, u1 = fifth-order
 * solution, err = |x_5 - x_4|; u1 normalised.  All pointers DEVICE; x3, u3, x1, u1 hold 3 n doubles (xyz per state).  EMX_E_STATE
 * when no field is set. */
int emx_field_substep_batch(emx_problem *p, long n, const double *x3, const double *u3, const double *kappa,
                            const double *h, double *x1, double *u1, double *err, void *stream);

/* Level-1 parity hooks (integer work).  All pointers DEVICE.
 * emx_philox_batch: out[4i..4i+3] = Philox4x32-10(ctr[4i..], key[2i..]).
 * emx_draw_batch:   u[i] = draw number n[i] of (seed, prim[i], tid[i], step[i]); child[i] = child track id
 *                   for ordinal n[i] (either output may be NULL). */
int emx_philox_batch(long n, const uint32_t *ctr4, const uint32_t *key2, uint32_t *out4, void *stream);
int emx_draw_batch(uint64_t seed, long n, const uint32_t *prim, const uint64_t *tid, const uint32_t *step,
                   const uint32_t *nn, double *u, uint64_t *child, void *stream);

/* Level-1 hook for the relocation after a boundary crossing (C8; HOST only, needs no device and no
 * tables): the candidate cells, in the order they are tested, for a track that has crossed `surface` towards
 * its `sense` side (+1: f > 0, -1: f < 0).  which = 0: the cells that list (surface, sense); which = 1: the cells
 * that do not list the surface at all.  Both lists leave out the cells a parallel face of their own keeps on the
 * other side of the surface by more than max(1e-6 cm, 10 field_eps).  Writes min(count, cap) cell ids to
 * host_out (may be NULL with cap = 0) and returns count, or EMX_E_ARG. */
int emx_neighbour_candidates(const emx_problem *p, int surface, int sense, int which, int32_t *host_out, int cap);

/* Level-1 hook for the refill / compaction step: applies one refill pass to a pool
 * of `n_live` slots whose alive flags are alive[n_live] (uint8, DEVICE) with `n_queue` queued records and
 * room for `capacity` slots, and writes, for every slot index < new_n_live, src[i] (int32, DEVICE,
 * capacity entries): -1 = untouched live track, q >= 0 = filled from queue record q,
 * -2 - j = moved from slot j.  counts_host[3] = { new_n_live, new_n_queue, holes the stack could not
 * fill (= old n_live - new n_live when positive) }. */
int emx_refill_plan(long n_live, long capacity, long n_queue, const uint8_t *alive, int32_t *src,
                    long *counts_host, void *stream);

/* The same hook for callers that may not allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): identical arguments and results, but the scratch of the refill kernels
 * (chunk tables, hole list, control block, a padded copy of alive[]) lives in a file-scope device array of the
 * library instead of a block that emx_refill_plan allocates and frees on every call.  The call allocates nothing:
 * no cudaMalloc, cudaFree or allocating library routine, on the host or on the device.
 *   limit       capacity <= emx_refill_plan_static_max() = 65536 slots; a larger capacity returns EMX_E_CAPACITY
 *               with a text naming the limit (use emx_refill_plan there).  The array is 345 KB; every GPU that loads
 *               the library holds it until the process exits.
 *   set-up      the device address of the array is looked up once per device (cudaGetSymbolAddress with that device
 *               current) on the first call there; emx_refill_plan_static_setup() does the lookup for the current
 *               device ahead of time and returns EMX_OK or EMX_E_CUDA / EMX_E_ARG (device ordinal above 63).
 *   sharing     every call on a device uses the SAME array.  It keeps the previous call's contents, so each call
 *               clears the part it uses first (on `stream`).  Calls whose GPU work overlaps -- different streams,
 *               or different host threads -- race on it: serialise them.  Calls on one stream are safe, and the
 *               function returns only after its own work on `stream` is complete.
 * alive, src: DEVICE, owned by the caller; counts_host: HOST. */
int emx_refill_plan_static(long n_live, long capacity, long n_queue, const uint8_t *alive, int32_t *src,
                           long *counts_host, void *stream);
long emx_refill_plan_static_max(void);
int emx_refill_plan_static_setup(void);

const char *emx_last_error(const emx_problem *p);
const char *emx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EMX_H */
