/*
 * genga.h -- C-ABI of the B200-native hybrid symplectic integrator
 * (Grimm & Stadel, "The GENGA code", arxiv 1404.2324; line numbers refer to PAPER.md).
 *
 * One context = one simulation in one of the paper's three modes:
 *   mode 0  up to 2048 massive bodies about one central mass,
 *   mode 1  up to 32 massive bodies plus up to 10^6 massless test particles (L334-342),
 *   mode 2  up to 100000 independent systems of up to 16 bodies each (L344-376).
 * Every step of the method runs in CUDA kernels on the stream given at creation; this
 * library never falls back to the CPU.  It needs an sm_100a device.
 *
 * Body layout (all modes): SoA, Ntot = n_massive + n_test (modes 0,1) or
 * n_systems * n_massive (mode 2; body index = system * n_massive + k).
 * 3-vectors are stored as x[c * Ntot + i], c = 0,1,2.  Massive bodies come first.
 *
 * Coordinates at the boundary are HELIOCENTRIC positions and HELIOCENTRIC velocities;
 * internally the integrator works in democratic coordinates (heliocentric positions,
 * barycentric velocities, L69).  Units: whatever makes G the value given in the config
 * (G = 1 with AU, M_sun, day/k).
 *
 * Ownership: the caller owns every buffer, including the workspace and the stream; the
 * context owns only a small host structure.  "device" / "host" below says where a
 * pointer must point.  Buffers passed to a call may be reused once the work the call
 * enqueued has completed on the stream (the *_host variants and genga_energy /
 * genga_encounters / genga_status synchronise the stream before returning).
 *
 * Errors: every call returns 0 or a negative genga_error.  Conditions detected on the
 * device during genga_step (Kepler or Bulirsch-Stoer non-convergence, pair list
 * overflow) are latched in a device word and returned by the next synchronising call
 * (genga_status, genga_get_state_host, genga_energy, genga_encounters).
 */
#ifndef GENGA_H
#define GENGA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct genga_ctx genga_ctx;

typedef enum {
    GENGA_OK = 0,
    GENGA_EINVAL = -1,    /* bad mode / sizes / order / dt == 0 / NULL pointer / workspace too small */
    GENGA_ECAPACITY = -2, /* candidate or encounter pair list exceeded max_pairs */
    GENGA_EKEPLER = -3,   /* universal-variable Kepler solver did not converge */
    GENGA_EBS = -4,       /* Bulirsch-Stoer step size underflow */
    GENGA_ECUDA = -5      /* a CUDA runtime call failed (see genga_last_cuda_error) */
} genga_error;

enum { GENGA_MODE_MASSIVE = 0, GENGA_MODE_TEST_PARTICLE = 1, GENGA_MODE_MULTI_SYSTEM = 2 };

typedef struct {
    int32_t mode;       /* GENGA_MODE_*                                                      */
    int32_t n_massive;  /* per system: 1..2048 (mode 0), 1..32 (mode 1), 1..16 (mode 2); L188  */
    int64_t n_test;     /* mode 1 only: 0..10^6 test particles; else 0                        */
    int32_t n_systems;  /* mode 2 only: 1..100000; else 1                                     */
    int32_t flags;      /* bit 0: do not merge the closing kick of a substep with the opening kick
                           of the next substep of the same step (orders 4, 6; modes 0, 2; L170);
                           the result is the same map, this only selects the schedule;
                           bit 1: mode 0, do not reuse the far-pair sums of a step's closing kick in the
                           opening kick of the next step (L266-274); same map, schedule only;
                           bit 2: mode 2, run a step as one launch per operator over all systems instead of
                           one launch per call in which every block runs its own systems ahead          */
    double G;           /* gravitational constant                                            */
    double n1, n2;      /* critical-radius parameters of Eq. 6 (L94-96); usually 3 and 0.4   */
    double bs_eps;      /* Bulirsch-Stoer relative tolerance (L116 "machine precision")      */
    int64_t max_pairs;  /* capacity of the candidate list and of the encounter list, 1 .. 2^31 - 1 */
    void *workspace;    /* device memory, >= genga_workspace_bytes(), 256-byte aligned        */
    size_t workspace_bytes;
    void *stream;       /* cudaStream_t; NULL = the legacy default stream                     */
} genga_config;

/* Bytes of device workspace a context with this config needs (workspace fields ignored).
 * Returns 0 if the config is invalid. */
size_t genga_workspace_bytes(const genga_config *cfg);

/* Create / destroy a context.  genga_create does not touch the device state arrays;
 * call genga_set_state before anything else. */
/* Environment: GENGA_NO_PDL=1 (read by genga_create) launches the kernels of a step without programmatic
 * dependent launch; GENGA_TMA=1 makes the pair kernel of the kick stage the records of its partner tile with bulk copies
 * (cp.async.bulk + one mbarrier per slice) instead of through registers (measured on B200 at N = 2048: 12.4 against
 * 11.7 us per launch, so it is not the default); results are bit-identical either way. */
int genga_create(const genga_config *cfg, genga_ctx **out);
int genga_destroy(genga_ctx *ctx);

/* Load the state (problem statement: L69, L188, L316-324, L352).
 *   m0[n_systems]  central masses; m[Ntot] masses (0 for test particles); radius[Ntot]
 *   physical radii (used once genga_set_collisions switches collisions on); x[3*Ntot], v[3*Ntot]
 *   heliocentric positions / velocities.
 * genga_set_state: all pointers DEVICE.  genga_set_state_host: all pointers HOST (pinned
 * or pageable); the copies are enqueued on the stream and the call returns after they and
 * the conversion to democratic coordinates have completed.  States of up to 512 KB (and a
 * non-NULL radius) are packed into a pinned image owned by the context and moved with ONE
 * copy (genga_get_state_host likewise), and the call returns as soon as the caller's
 * buffers have been read, the copy still in flight on the stream; larger ones are copied
 * array by array straight from the caller's buffers. */
int genga_set_state(genga_ctx *ctx, const double *m0, const double *m, const double *radius,
                    const double *x, const double *v);
int genga_set_state_host(genga_ctx *ctx, const double *m0, const double *m, const double *radius,
                         const double *x, const double *v);

/* The kernel sequence of (dt, order) is captured into CUDA graphs (16 steps, 1 step) the first time it is used and
 * replayed afterwards; the cache is keyed on the exact value of dt and holds 16 entries (a 17th clears it), so a
 * caller that changes dt at every call pays a capture (~1 ms) per call.
 * Advance n_steps time steps of length dt (dt < 0 integrates backwards) with the hybrid
 * symplectic scheme of order 2 (Eq. 7; per-step algorithm), 4 or 6
 * (Yoshida compositions, L168-170).  Each step: critical radii (Eq. 6), kick with the
 * changeover weight and prechecker (Eq. 2), Sun kick (Eq. 3), Kepler drift (Eq. 9),
 * encounter search (Eq. 10-12), grouping (Appendix), Bulirsch-Stoer on the groups (L116),
 * Sun kick, kick.  Work is enqueued on the stream; the call does not synchronise. */
int genga_step(genga_ctx *ctx, int64_t n_steps, double dt, int order);

/* Read the state back as heliocentric x[3*Ntot], v[3*Ntot].  DEVICE pointers (enqueued,
 * no sync) or HOST pointers (synchronises; returns a latched device error if any). */
int genga_get_state(genga_ctx *ctx, double *x, double *v);
int genga_get_state_host(genga_ctx *ctx, double *x, double *v);

/* Multi-system mode with a VARIABLE number of bodies per system (L346-354: "no more than 16
 * bodies" each).  System s holds n_bodies[s] bodies, 1 <= n_bodies[s] <=
 * n_massive; the packed arrays list the systems one after the other (start index of system
 * s = sum of n_bodies[0..s-1], Nreal = sum of all): m[Nreal], radius[Nreal] (may be NULL),
 * x[3*Nreal] = all x, all y, all z, v likewise; m0[n_systems].  HOST pointers.
 * Inside, every system keeps n_massive slots (body = system * n_massive + k); the unused slots
 * hold MASSLESS bodies on wide circular orbits (1000 (k + 1) length units from the central
 * mass): they exert no force, add exact zeros to every sum, never come within a critical
 * radius of anything, so the real bodies move exactly as in a system of n_bodies[s] slots.
 * The other calls keep the padded indexing (genga_get_state*, genga_encounters labels);
 * genga_get_state_ragged_host returns the real bodies in the packed order.  Both synchronise.
 * GENGA_EINVAL outside multi-system mode, for a size out of range, or (get) before a set. */
int genga_set_state_ragged_host(genga_ctx *ctx, const int32_t *n_bodies, const double *m0, const double *m,
                                const double *radius, const double *x, const double *v);
int genga_get_state_ragged_host(genga_ctx *ctx, double *x, double *v);

/* Multi-system mode: the n1 and n2 of Eq. 6 (L94-96) of every system (L346-354: among the few
 * parameters that "can be set individually for the different simulations"; the central mass
 * is m0[] of genga_set_state).  n1[n_systems], n2[n_systems], HOST pointers, both >= 0; they
 * replace the configuration's values from the next step on.  Synchronises.  GENGA_EINVAL
 * outside multi-system mode. */
int genga_set_system_params_host(genga_ctx *ctx, const double *n1, const double *n2);

/* Total energy E[n_systems] and angular momentum L[3*n_systems] (x,y,z per system) of the
 * current state, Eq. 1-3 summed (L73-80).  HOST pointers; synchronises.  L may be NULL. */
int genga_energy(genga_ctx *ctx, double *E, double *L);

/* Close-encounter data of the LAST drift substep executed (L118-142, L276-284):
 *   pairs[2*cap]  confirmed pairs (i, j), i < j, global body indices, sorted by (i, j);
 *                 at most cap are written;   *n_pairs = number confirmed;
 *   *n_candidates = number of prechecker candidates of that substep;
 *   group_label[Ntot] (or NULL): lowest body index of the body's encounter group, the
 *                 body's own index if it is in no group.
 * HOST pointers; synchronises. */
int genga_encounters(genga_ctx *ctx, int32_t *pairs, int64_t cap, int64_t *n_pairs,
                     int64_t *n_candidates, int32_t *group_label);

/* Collisions, ejections and removal of bodies (L316-332 sections 3.2.7-3.2.8, L336, L378-384; SURVEY 8(f) NEXT-1..3).
 * Off after genga_create: bodies are point masses.  genga_set_collisions switches on
 *   collisions != 0: between the Bulirsch-Stoer steps of every group the minimum of the cubic Hermite interpolant of the
 *     squared separation over the step (Eq. 10-12; "the same code as in the close encounter detection", L328) is compared
 *     with (R_i + R_j)^2.  A colliding pair merges as perfectly inelastic bodies at the end of that step: mass and linear
 *     momentum conserved, position = centre of mass, radius (R_i^3 + R_j^3)^(1/3), internal energy U += 1/2 m_i m_j /
 *     (m_i + m_j) v_ij^2 - G m_i m_j / r_ij (L318-322), spin from angular momentum conservation, the new body keeps the
 *     index of the more massive one (the smaller index if equal); the other becomes a massless ghost parked on a
 *     circular orbit of radius 1000 (k + 1) (k = its index within its system), where it meets nothing and adds exact
 *     zeros to every sum -- "removed later" (L324): the caller compacts by reloading the state without the removed
 *     bodies.  A test particle that hits a massive body is reported and removed, with no effect on the body (L336).
 *   rcut, rcut_sun > 0: at the end of a time step a body farther from the central mass than rcut, or closer than
 *     rcut_sun, is reported and removed (L330-332).
 *   n_min > 0: a system with fewer than n_min massive bodies left is stopped: all its bodies are removed (L378-384).
 * Synchronises; drops the cached CUDA graphs.
 * genga_events: the records since the last genga_set_state*, at most 4096 are kept; *n = number made.  A record is 24
 * doubles: [0] steps completed before the event's step, [1] kind (0 collision, 1 test particle hit a massive body,
 * 2 beyond rcut, 3 inside rcut_sun, 4 removed because its system stopped), [2] surviving body (or the body removed by
 * kinds 2-4), [3] removed body (-1 for kinds 2-4), [4..5] masses, [6..7] radii, [8..10], [11..13] heliocentric position
 * and BARYCENTRIC velocity of body [2] at the start of the Bulirsch-Stoer step in which the collision happened ("the
 * last time step before the collision", L326; kinds 2-4: at the end of the step), [14..19] the same of body [3],
 * [20] the internal energy of this collision, [21..23] spin of the new body.  Order of the records: not defined.
 * genga_bodies: current m[Ntot], radius[Ntot], kind[Ntot] (0 massive, 1 test particle, 2 removed), spin[3*Ntot],
 * U[n_systems]; any pointer may be NULL.  HOST pointers; both synchronise. */
int genga_set_collisions(genga_ctx *ctx, int collisions, double rcut, double rcut_sun, int n_min);
int genga_events(genga_ctx *ctx, double *records, int64_t cap, int64_t *n);
int genga_bodies(genga_ctx *ctx, double *m, double *radius, int32_t *kind, double *spin, double *U);

/* One record per encounter group that Bulirsch-Stoer integrated in the LAST drift substep executed (L116, L286-314;
 * at most 4096 are kept): out[4*k + 0] = group size | layout << 16 (layout 0: one warp, 1: cluster),
 * out[4*k + 1] = accepted steps | rejected attempts << 16, out[4*k + 2] = SM clock cycles the integration took,
 * out[4*k + 3] = a member's body index.  *n = number of records made (may exceed cap and 4096).  The step time of an
 * encounter-heavy run is the longest of these chains; bench.py reports it.  HOST pointers; synchronises. */
int genga_bs_trace(genga_ctx *ctx, int32_t *out, int64_t cap, int64_t *n);

/* Synchronise the stream and return (and clear) the latched device error, or GENGA_OK. */
int genga_status(genga_ctx *ctx);

/* ---- auxiliary entry points: single operators of the path, for tests and kernel timing ---- */

/* Critical radii for a step dt at the current state (Eq. 6) and the kick accelerations
 * a[3*Ntot] of operator B there (Eq. 2 with the changeover weight); also refreshes the
 * candidate list.  a, rcrit DEVICE pointers (rcrit may be NULL).  Enqueues, no sync. */
int genga_accelerations(genga_ctx *ctx, double dt, double *a, double *rcrit);

/* Kepler drift (Eq. 9, universal variables) of n independent bodies about mu for time h:
 * x[3*n], v[3*n] DEVICE, updated in place.  Stand-alone: needs no state in the context. */
int genga_kepler_drift(genga_ctx *ctx, int64_t n, double mu, double h, double *x, double *v);

/* Counters accumulated since genga_create, HOST out[16]:
 *  0 steps, 1 force evaluations, 2 ordered pair interactions evaluated, 3 kernel launches,
 *  4 groups integrated, 5 largest group, 6 BS steps accepted, 7 candidates seen,
 *  8 BS attempts rejected (all eight extrapolation columns failed, step halved), 9..15 reserved (0).
 * Synchronises. */
int genga_counters(genga_ctx *ctx, int64_t *out);

/* Time one kernel of the path in isolation on the context's stream with CUDA events:
 * `reps` back-to-back launches after 3 warm-up launches, *ms_per_launch = average (HOST out).
 *   which = 0  pair kernel of the kick (k_kick; modes 0, 1), current state and rcrit
 *   which = 1  Kepler drift of all bodies over dt and back (two launches counted as two)
 *   which = 2  the whole kick (k_kick [+ k_tp_kick of the test particles]), h = 0
 *   which = 3  mode 1: fused particle pass kick + Sun kick + drift (k_tp_front) over dt and back
 *   which = 4  mode 1: fused particle pass Sun kick + kick (k_tp_back) over dt and back
 *   which = 5  mode 1: closing half + opening half + drift + encounter search in one pass (k_tp_mid) over dt and back
 * The state is left unchanged up to rounding (3, 4: up to the integration error of the
 * pass and its inverse).  Synchronises. */
int genga_time_kernel(genga_ctx *ctx, int which, int reps, double dt, double *ms_per_launch);

/* Run n_steps (1..4096) time steps exactly as genga_step does, but as plain launches with a CUDA event at every
 * phase boundary instead of a graph replay, and report the time per step of each phase, HOST ms[8]:
 *   0 critical radii (Eq. 6)   1 kicks (Eq. 2; every pair-force launch of the step)
 *   2 opening half map: Sun kick + Kepler drift (Eq. 3, Eq. 9; the fused half-map kernels of the small-N,
 *     particle and multi-system layouts count here as a whole, their kick included)
 *   3 encounter search (Eq. 10-12)   4 grouping (Appendix)   5 Bulirsch-Stoer (L116), all layouts
 *   6 closing half map: Sun kick (and kick where fused)   7 sum of the phases.
 * The state advances by n_steps steps.  Synchronises. */
int genga_profile_step(genga_ctx *ctx, int64_t n_steps, double dt, int order, double *ms);

/* out[i] = f(in[i]) with the library's reciprocal routines built on the hardware seeds, in FP64:
 * which = 0: x^(-1/2), 1: x^(-3/2), 2: 1/x, for positive normal x.  The paper keeps IEEE sqrt and divide for fear of a
 * biased error (L228, L264); tests/test_gpu_fastmath.py measures the signed error of these in ulps.
 * in, out: DEVICE pointers to n doubles.  Enqueues, no sync. */
int genga_eval_fast(genga_ctx *ctx, int which, int64_t n, const double *in, double *out);

/* Measure the device's FP64 FMA throughput with independent DFMA chains on every SM:
 * *tflops (HOST out) = 2 * DFMAs / time.  The ALU-roofline denominator.  Synchronises. */
int genga_fp64_probe(genga_ctx *ctx, double *tflops);

/* ---- an entry point that allocates nothing (csrc/noalloc.cu) ----
 * Kick accelerations of operator B for ONE system of n massive bodies, without a context and without a workspace:
 * a_i = sum_{j != i} G m_j W(r_ij, max(rcrit_i, rcrit_j)) (q_j - q_i) / r_ij^3, W = K - r dK/dr (Eq. 2, Eq. 4-8
 * L84-104): what genga_accelerations returns in `a` for the same positions, masses and critical radii (to rounding:
 * the partial sums are added in another order).  For callers that cannot call cudaMalloc (CUDA graph capture, serving
 * loops, harnesses that forbid it): the kernels' scratch memory (packed body records, partial sums of 16 j slices) is
 * a file-scope device array of GENGA_NOALLOC_SCRATCH_BYTES that every GPU which loads the library holds until the
 * process exits; the call makes no cudaMalloc, cudaFree or other allocating call and does not synchronise.
 *   stream      cudaStream_t (may be 0); three kernels are enqueued on it
 *   n           0 .. GENGA_NOALLOC_MAX_BODIES; a larger n is rejected with GENGA_EINVAL (genga_noalloc_last_error says why)
 *   G           > 0
 *   m, rcrit    DEVICE, n doubles each; x DEVICE, 3 n doubles, component-major (x[c * n + i]); owned by the caller, read only
 *   a           DEVICE out, 3 n doubles, component-major
 * All calls on one device SHARE the scratch array, which keeps the last call's contents; a call writes every word it
 * reads, so nothing needs clearing, but two calls that overlap on the GPU (different streams, concurrent graph
 * launches) race: serialise them.  Returns GENGA_OK, GENGA_EINVAL (sizes, NULL, G) or GENGA_ECUDA. */
#define GENGA_NOALLOC_MAX_BODIES 2048
#define GENGA_NOALLOC_SCRATCH_BYTES 868352
int genga_kick_accel_noalloc(void *stream, int64_t n, double G, const double *m, const double *x, const double *rcrit, double *a);
/* The reason of the last GENGA_EINVAL / GENGA_ECUDA of genga_kick_accel_noalloc on this thread ("" if none). */
const char *genga_noalloc_last_error(void);

const char *genga_strerror(int code);
const char *genga_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GENGA_H */
