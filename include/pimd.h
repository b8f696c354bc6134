/*
 * pimd.h -- C ABI of libpimd.so: the per-time-step force evaluation and the thermostatted
 * velocity-Verlet update of bosonic / xi-particle path integral molecular dynamics as defined
 * in arXiv 2404.02628 (cited as PAPER.md:<line>, Eq. <n>), hand-written CUDA for sm_100a.
 *
 * What is computed (units hbar = m = k_B = 1):
 *   sampled potential  Phi = V_xi^{[1,N]} + U/P                       (Eq. 4)
 *   V_xi^{[1,N]}       by the recursion of Eq. 6 over the cycle energies of
 *                      Eq. 7, spring constant k_s = m omega_P^2 = P/beta^2
 *   U                  sum_j [ sum_l 1/2 omega^2 |r_l^j|^2 + sum_{i<l} g exp(-|r_l^j-r_i^j|^2/s^2) ]
 *                      (Eq. 5 :55, Eq. 18 :142, Eq. 19 :158, Eq. 20 :193 with g = g_paper/(pi s^2))
 *   forces             F = -grad Phi: Eq. 15, 16 (beads 1 and P, through the connection
 *                      probabilities of Eq. 12-14), Eq. 17 (interior beads, :136)
 *                      and -(1/P) grad U
 *   dynamics           velocity Verlet with a thermostat at T = 1/beta (R10)
 *
 * Conventions
 *   - Every function returns PIMD_OK (0) or a negative PIMD_E* code; pimd_last_error() gives text.
 *     No C++ type or exception crosses this boundary.
 *   - "dev" pointers are CUDA device pointers, "host" pointers are host pointers.  The caller owns
 *     every buffer it passes; the library copies in/out and never keeps a caller pointer, except
 *     the workspace given to pimd_set_workspace(), which the caller must keep alive until
 *     pimd_destroy() or the next pimd_set_workspace().
 *   - State layout: x[P][N][d], v[P][N][d], f[P][N][d], C-contiguous doubles, flat index
 *     ((j*N)+l)*d+c for bead j (0..P-1 <-> the paper's 1..P), particle l (0..N-1), coordinate c.
 *     Particle order is significant (the recursion threads cycles over consecutive indices).
 *   - All work is enqueued on the stream given by pimd_set_stream() (default: the legacy default
 *     stream) and on one internal helper stream that is fork/joined to it with events.  Calls that
 *     return host scalars synchronise that stream; pimd_step() is asynchronous.
 *   - One handle is not thread-safe; different handles are independent.
 *   - Environment knobs read by pimd_create() (tuning / debugging only): PIMD_LOOK (column blocks kept inside the
 *     chain CTA, 1..3), PIMD_WORKERS (panel worker CTAs per direction), PIMD_NOSPEC=1 (always run the max-plus
 *     recursion kernel, never the stale-gauge one), PIMD_PAIR_CH (tile offsets per pair-kernel task), PIMD_PAIR2=0/1 (pair
 *     kernel with one / two row particles per lane instead of the choice by size: two from N = 1500 on), PIMD_GRAPH=0
 *     (pimd_step launches every kernel itself instead of replaying a captured CUDA graph).
 *   - There is no CPU fallback: without a CUDA device pimd_create() fails with PIMD_ECUDA.
 */
#ifndef PIMD_H
#define PIMD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PIMD_OK 0
#define PIMD_EINVAL (-1)   /* bad argument (N<1, P<2, d not in {1,2,3}, beta<=0, s<=0, dt<=0, non-finite, ...) */
#define PIMD_ENOMEM (-2)   /* host or device allocation failed / workspace too small */
#define PIMD_ECUDA (-3)    /* a CUDA call failed; pimd_last_error() holds the CUDA error string */
#define PIMD_ENUMERIC (-4) /* non-finite state, or e^{-beta V} summed to exactly zero (a node, xi<0) */

#define PIMD_THERMOSTAT_NVE 0      /* none */
#define PIMD_THERMOSTAT_LANGEVIN 1 /* OBABO, friction gamma (default 1), Philox4x32-10 noise */
#define PIMD_THERMOSTAT_NHC 2      /* massive Nose-Hoover chains, length 4, Q = beta/P */
#define PIMD_NHC_LENGTH 4
#define PIMD_MAX_SPECIES 4
#define PIMD_MAX_BINS 4096         /* histogram bins (radial density, pair distances) */
#define PIMD_PAIR_GAUSSIAN 0       /* v(r) = g exp(-r^2/s^2)      (Eq. 20, with g = g_paper/(pi s^2)) */
#define PIMD_PAIR_SOFT_COULOMB 1   /* v(r) = g / sqrt(r^2 + s^2)  (Eq. 18, leaves the pair potential open) */

typedef struct pimd_s *pimd_t; /* opaque; owns its device workspace unless one is supplied */

/* Create a simulation of N particles x P beads in d dimensions at inverse temperature beta in an
 * isotropic harmonic trap of frequency omega, pair potential g*exp(-r^2/s^2) between same-index
 * beads, exchange parameter xi (1 bosons, 0 distinguishable, <0 fictitious particles; Eq. 2,
 * PAPER.md:39-42), time step dt, thermostat PIMD_THERMOSTAT_*, noise seed.  State starts at zero;
 * load it with pimd_set_state().  *out is NULL on failure (then pimd_last_error(NULL) has text). */
int pimd_create(pimd_t *out, int N, int P, int d, double beta, double omega, double g, double s,
                double xi, double dt, int thermostat, uint64_t seed);
int pimd_destroy(pimd_t h);

/* A batch of B replicas of the same system that differ in the exchange parameter xi[b] and the noise seed[b] (HOST
 * arrays of B entries), advanced by one set of kernel launches (replica = a grid dimension).  This is how the method is
 * used for fictitious particles: simulate at several xi >= 0 and extrapolate / reweight; it also
 * fills the GPU at small N.  Either every xi[b] is 0 or none is.  With a batch every state / force array of this header
 * is [B][P][N][d] and every per-evaluation HOST output (vb, sign, e_prim, e_vir, hist, ...) has B entries (hist: [B][nbins]);
 * pimd_create() is the batch with B = 1.  B is limited by the CTAs of the recursion kernel that must be co-resident (one
 * 512-thread CTA per SM): 2 per replica while every species has at most 32*(PIMD_LOOK+1) = 128 particles, 4 per replica
 * (chain + at least one panel worker per direction) beyond that.  On a B200 (148 SMs): 74 replicas at N <= 128, 37 for
 * larger N; a larger batch is refused with PIMD_EINVAL (by pimd_create_batch, or by pimd_set_species if the species
 * partition is what needs the workers). */
int pimd_create_batch(pimd_t *out, int B, int N, int P, int d, double beta, double omega, double g, double s,
                      const double *xi, double dt, int thermostat, const uint64_t *seed);

/* Several species of identical particles (the spin-unpolarised case): particles [0, counts[0]) are species
 * 0, the next counts[1] species 1, ...; exchange (Eq. 6, 11-16) acts within a species only, V_xi = sum over species of
 * V_xi^{[range]}, the trap and pair terms act on all particles alike.  counts: HOST, nspecies <= PIMD_MAX_SPECIES
 * entries that add up to N.  Must precede the first state / compute call.  vb returned by pimd_forces is the sum over
 * species, sign the product. */
int pimd_set_species(pimd_t h, int nspecies, const int *counts);

/* Pair potential between same-index beads (Eq. 18): PIMD_PAIR_GAUSSIAN (default) or PIMD_PAIR_SOFT_COULOMB,
 * both with the g and s of pimd_create. */
int pimd_set_pair_potential(pimd_t h, int kind);

/* cuda_stream is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default. */
int pimd_set_stream(pimd_t h, void *cuda_stream);

/* Device workspace.  pimd_workspace_bytes() is the size needed; pimd_set_workspace() hands the
 * library caller-owned device memory (256-byte aligned, e.g. a torch uint8 tensor) to use instead
 * of its own cudaMalloc.  Must be called before the first compute/state call. */
size_t pimd_workspace_bytes(pimd_t h);
int pimd_set_workspace(pimd_t h, void *dev_ptr, size_t bytes);

/* Langevin friction gamma (>0; default 1).  Other thermostat parameters are fixed (R10). */
int pimd_set_gamma(pimd_t h, double gamma);
/* 1 (default): the exchange part and the pair part of a force evaluation run concurrently on two
 * streams; 0: everything on the main stream (profiling / debugging). */
int pimd_set_concurrency(pimd_t h, int on);

/* Copy state in / out.  x_dev, v_dev: DEVICE pointers, [P][N][d] doubles; v_dev may be NULL
 * (set: velocities zero; get: skipped).  Setting the state resets the Nose-Hoover variables to zero
 * and invalidates cached forces (see pimd_set_forces).  *_host variants take HOST pointers (pageable or pinned). */
int pimd_set_state(pimd_t h, const double *x_dev, const double *v_dev);
int pimd_get_state(pimd_t h, double *x_dev, double *v_dev);
int pimd_set_state_host(pimd_t h, const double *x_host, const double *v_host);
int pimd_get_state_host(pimd_t h, double *x_host, double *v_host);
/* Resume support: MD step counter (the Philox counter of the Langevin noise) and the Nose-Hoover
 * chain variables nhc[PIMD_NHC_LENGTH][P*N*d] (DEVICE pointer).  A run continued in a new handle from
 * (pimd_set_state, pimd_set_forces, pimd_set_step_count, pimd_set_nhc -- in this order: setting the state zeroes the chain
 * variables) draws the same noise and follows the original trajectory to rounding (1e-12 after 10 steps in the tests), not
 * to the bit: the new handle's first evaluation has no gauge history and the pair forces are accumulated with atomics. */
int pimd_get_step_count(pimd_t h, uint64_t *step_host);
int pimd_set_step_count(pimd_t h, uint64_t step);
int pimd_get_nhc(pimd_t h, double *nhc_dev);
int pimd_set_nhc(pimd_t h, const double *nhc_dev);

/* One force evaluation at the current positions (steps 1-6 of the hot path).
 *   f_dev  DEVICE [P][N][d] or NULL: F = -grad( V_xi^{[1,N]} + U/P )
 *   vb     HOST out or NULL: V_xi^{[1,N]} = -(1/beta) ln|W_N|              (Eq. 6)
 *   sign   HOST out or NULL: sign of W_N = e^{-beta V} (+1 whenever xi >= 0)
 * Synchronises the stream.  PIMD_ENUMERIC if the state is non-finite or W_N == 0. */
int pimd_forces(pimd_t h, double *f_dev, double *vb, int *sign);
int pimd_forces_host(pimd_t h, double *f_host, double *vb, int *sign);

/* Cached total forces F = -grad(V_xi + U/P) at the current positions, [P][N][d] (DEVICE / HOST variants).
 * get: no evaluation is made; PIMD_EINVAL if no forces are cached (state just set, nothing evaluated).  Synchronises.
 * set: hands the library the forces that belong to the state just set with pimd_set_state() (checkpoint resume,
 * host-resident states), so that the next pimd_step() does not have to evaluate them first.  The caller vouches for
 * them; call after pimd_set_state(). */
int pimd_get_forces(pimd_t h, double *f_dev);
int pimd_get_forces_host(pimd_t h, double *f_host);
int pimd_set_forces(pimd_t h, const double *f_dev);
int pimd_set_forces_host(pimd_t h, const double *f_host);

/* Tables of the last force evaluation, HOST out (any may be NULL):
 *   vfwd[n] = V_xi^{[1,n]}, n = 0..N  (N+1 doubles; Eq. 6)
 *   vbwd[u] = V_xi^{[u,N]}, u = 1..N+1 stored at index u (N+2 doubles, index 0 unused; Eq. 11)
 *   pnext[l] = Pr[G(l) = l+1], l = 1..N stored at l-1 (N doubles; Eq. 13). */
int pimd_get_tables(pimd_t h, double *vfwd, double *vbwd, double *pnext);
/* A diagnostic call, not part of the hot path: the device holds the tables as per-block gauges plus residuals; this call
 * copies them out and finishes vfwd / vbwd with HOST arithmetic (long double prefix sums) inside the library. */

/* The paper's N x N intermediates, materialised on request into caller memory (DEVICE, N*N doubles, row-major;
 * the hot path never stores them).  Both synchronise.  N <= 65535.
 *   pimd_cycle_energies:            e[u*N + v] = E^{[u+1,v+1]} for u <= v (Eq. 7-10), 0 below the
 *                                   diagonal; computed from the current positions alone.
 *   pimd_connection_probabilities:  pr[l*N + m] = Pr[G(l+1) = m+1] (Eq. 12-14); signed
 *                                   quasi-probabilities for xi < 0, the identity for xi = 0.  Uses the tables of the
 *                                   last force evaluation at the current positions (evaluates first if there is none). */
int pimd_cycle_energies(pimd_t h, double *e_dev);
int pimd_connection_probabilities(pimd_t h, double *pr_dev);

/* The cycle energies of Eq. 7-10 without a handle and without any allocation.
 *
 * Who this is for.  Every other compute call of this header needs a handle, and making a handle allocates: device memory
 * for the workspace (cudaMalloc, unless pimd_set_workspace supplies it), pinned host memory, streams and events.  Some
 * programs cannot afford that at the point where they need the result:
 *   - a host application (an MD driver, a Python framework with a caching allocator) that has already claimed all the
 *     device memory it is allowed to use, so that a cudaMalloc made behind its back fails or pushes it over its budget;
 *   - a time-step loop with several streams in flight: cudaMalloc and cudaFree make the whole device wait, every stream
 *     stalls and the overlap the loop was built for is gone;
 *   - a plug-in or callback that runs where its host forbids allocation calls (a fixed memory plan made at start-up).
 * Such a caller passes only its own input and output buffers; the four O(N) intermediate tables (E_int, the closing
 * springs beta C(l,l+1) and their prefix sums S, T) live in a fixed array inside the library image, which the CUDA driver
 * places on each GPU when the library is loaded there and keeps until the process exits: 4 x PIMD_NOALLOC_MAX_N doubles =
 * 512 KiB per GPU, whether or not this function is ever called.
 *
 *   cuda_stream  cudaStream_t to enqueue on (NULL = default stream).  The call is ASYNCHRONOUS: it enqueues three kernels
 *                and returns; the result is complete when the stream reaches that point.
 *   x_dev        DEVICE in, [P][N][d] doubles, the state layout of this header; 16-byte aligned.  Not modified.
 *   N, P, d      1 <= N <= PIMD_NOALLOC_MAX_N, P >= 2, d in {1,2,3};  beta > 0 (k_s = P/beta^2 as everywhere here).
 *   e_dev        DEVICE out, N*N doubles, row-major: e[u*N + v] = E^{[u+1,v+1]} for u <= v, 0 below the diagonal
 *                (same contents as pimd_cycle_energies).
 * Returns PIMD_OK, or PIMD_EINVAL (bad argument; N > PIMD_NOALLOC_MAX_N is refused with a message that says so, nothing
 * is launched) or PIMD_ECUDA; text through pimd_last_error(NULL).
 *
 * Rules that follow from the shared array:
 *   - The first call on each device looks up the device address of the array (cudaGetSymbolAddress with that device
 *     current; it allocates nothing, but it may make the runtime load the library's kernels onto the device).  Make that
 *     first call during set-up, before any stream capture is begun.  Later calls on the device reuse the address.
 *   - The array is one per GPU, not per call or per stream, and keeps what the last call left in it.  A call writes every
 *     table entry before reading it, so stale contents are harmless, but two calls that can run on the GPU at the same
 *     time (different streams, or two host threads) overwrite each other's tables and both results are garbage.  Calls
 *     enqueued on one stream are ordered and safe.
 *   - The device that is current when the call is made must be the one that x_dev, e_dev and the stream belong to. */
#define PIMD_NOALLOC_MAX_N 16384
int pimd_cycle_energies_noalloc(void *cuda_stream, const double *x_dev, int N, int P, int d, double beta, double *e_dev);

/* Advance nsteps MD steps (asynchronous on the stream):
 *   thermostat half step ; v += dt/2 F ; x += dt v ; F = F(x) ; v += dt/2 F ; thermostat half step
 * Forces of the starting state are evaluated first if they are not cached.  For nsteps >= 3 (profiling off) all
 * but the last step replay one captured CUDA graph on an internal stream that is event-ordered with the caller's. */
int pimd_step(pimd_t h, int nsteps);

/* Estimators at the current positions (R9, R15), HOST outputs:
 *   e_prim = P d N/(2 beta) - <E_c> + Ubar   (thermodynamic estimator, -d ln Z/d beta of Eq. 4)
 *   e_vir  = Ubar + 1/2 sum r.grad Ubar       (virial estimator; valid in the trap)
 *   hist[b], b < nbins <= PIMD_MAX_BINS: number of beads with |r| in [b, b+1) * rmax/nbins (raw counts as doubles;
 *   beads with |r| >= rmax are dropped).  nbins may be 0 (hist ignored).  Synchronises. */
int pimd_estimators(pimd_t h, double *e_prim, double *e_vir, double *hist, int nbins, double rmax);

/* pimd_step with sampling: every step whose number (pimd_get_step_count after it) is a multiple of est_every > 0 makes
 * its force evaluation in estimator mode and adds e_prim, e_vir, the radial histogram (nbins bins on [0, rmax)) and the
 * pair-distance histogram (if pimd_set_pair_histogram is on) to running sums on the device.  Asynchronous; no extra
 * force evaluation is made for the estimators.  pimd_read_accumulators() synchronises and returns, per replica, the
 * number of samples and the sums (HOST; any pointer may be NULL; hist_sum [B][nbins], gr_sum [B][nbins_gr]); reset != 0
 * clears them afterwards. */
int pimd_run(pimd_t h, int nsteps, int est_every, int nbins, double rmax);
int pimd_read_accumulators(pimd_t h, double *nsamples, double *sum_eprim, double *sum_evir, double *hist_sum, int nbins,
                           double *gr_sum, int nbins_gr, int reset);

/* Pair-correlation estimator: histogram of the distances |r_l^j - r_i^j|, i < l, over all bead indices j (the pairs
 * Eq. 18, couples), nbins <= PIMD_MAX_BINS equal bins on [0, rmax), raw counts (normalisation by the caller).
 * Once switched on (nbins > 0) every estimator evaluation (pimd_estimators, sampling steps of pimd_run) fills it;
 * pimd_pair_histogram() returns the one of the last estimator evaluation (HOST, [B][nbins]). */
int pimd_set_pair_histogram(pimd_t h, int nbins, double rmax);
int pimd_pair_histogram(pimd_t h, double *gr_host);

/* Reweighting to a second exchange parameter (R7): the recursion of Eq. 6 is
 * evaluated at the current positions with xi_obs[b] (HOST, B entries) beside the sampling xi.  HOST outputs, B entries
 * each, any may be NULL:
 *   ln_abs_r = ln |W_{xi_obs} / W_{xi}| = -beta (V_{xi_obs} - V_{xi}),  sign = sign of that ratio,
 *   eps_obs, eps_samp = d(beta V)/d beta = -<E_c> at xi_obs / at the sampling xi,
 * so that the primitive energy estimator at xi_obs is e_prim (of pimd_estimators) - eps_samp + eps_obs and an observable O
 * at xi_obs is <O R> / <R> with R = sign exp(ln_abs_r) over a run at the sampling xi.  Synchronises.  PIMD_ENUMERIC if
 * W_{xi_obs} is exactly zero. */
int pimd_reweight(pimd_t h, const double *xi_obs, double *ln_abs_r, int *sign, double *eps_obs, double *eps_samp);

/* Bead shards (multi-GPU, one process per GPU).  Rank `rank` of `world` holds the bead slices
 * [floor(P rank/world), floor(P (rank+1)/world)) of every ring polymer: its state / force arrays are [P_local][N][d].
 * Springs, trap, pair forces, integrator and the bead sums of the estimators are local; the exchange part (steps 3-6,
 * O(N^2) against O(P N^2 / world) for the pair part) runs redundantly on every rank.  One exchange step per MD step: the
 * all-gather (by the caller: NCCL through torch.distributed, or a device copy between shards on one GPU) of every
 * rank's boundary pack of `pack_doubles` = 2 N d + N doubles, rounded up to an even count:
 *     [ first local slice : N d ][ last local slice : N d ][ E_int of the springs between local slices : N ].
 *   pimd_shard_export(h, send_dev)          write this rank's pack (DEVICE out); asynchronous
 *   pimd_shard_forces(h, gathered_dev)      take the gathered packs (DEVICE, world * pack_doubles, rank-major; copied)
 *                                           and evaluate the forces of the local slices; asynchronous
 *   pimd_shard_begin_step(h, send_dev)      thermostat half ; v += dt/2 F ; x += dt v ; export
 *   pimd_shard_end_step(h, gathered_dev)    import ; forces ; v += dt/2 F ; thermostat half
 *   pimd_shard_scalars(h, vb, sign)         V_B and sign of the last pimd_shard_forces (HOST; synchronises)
 * pimd_get_forces / pimd_get_state / pimd_set_state act on the local slices.  pimd_estimators on a shard returns this
 * rank's share (the bead sums over its slices; the kinetic constant and <E_c> on rank 0 only): the sum over ranks is the
 * estimator.  The Langevin noise of a degree of freedom is keyed by its global index, so a sharded run reproduces the
 * single-GPU trajectory.  pimd_forces, pimd_step, pimd_run, pimd_reweight refuse a shard (PIMD_EINVAL). */
int pimd_create_sharded(pimd_t *out, int rank, int world, int N, int P, int d, double beta, double omega, double g, double s,
                        double xi, double dt, int thermostat, uint64_t seed);
int pimd_shard_layout(pimd_t h, int *j0, int *p_local, size_t *pack_doubles);
int pimd_shard_export(pimd_t h, double *send_dev);
int pimd_shard_forces(pimd_t h, const double *gathered_dev);
int pimd_shard_begin_step(pimd_t h, double *send_dev);
int pimd_shard_end_step(pimd_t h, const double *gathered_dev);
int pimd_shard_scalars(pimd_t h, double *vb, int *sign);

/* Diagnostics (HOST out, 4 entries; synchronises): [0] force evaluations since creation in which the recursion with the
 * previous evaluation's gauge was rejected and redone with a fresh max-plus gauge, [1] PIMD status bits (1 non-finite,
 * 2 node) seen in any evaluation since the last pimd_set_state, [2] panel worker CTAs per direction, [3] bytes between
 * replicas in the workspace. */
int pimd_get_diagnostics(pimd_t h, uint64_t *out);

/* Device time of the kernels of the last pimd_forces()/pimd_step() force evaluation is not
 * recorded here; use CUDA events on the stream.  The number of kernel launches issued by the
 * library since creation (for bench.py's gpu_launches): */
uint64_t pimd_launch_count(pimd_t h);

/* Per-kernel device time.  With profiling on, every kernel launch is bracketed by a pair of CUDA
 * events on the stream it is launched on.  pimd_get_profile() synchronises, adds up the elapsed
 * times per slot since the previous call (milliseconds, and launch counts), returns them in the
 * HOST arrays ms_host / count_host (PIMD_PROF_NSLOTS entries each; either may be NULL) and resets. */
#define PIMD_PROF_BEAD 0      /* spring + trap forces (step 1) */
#define PIMD_PROF_PREP 1      /* closing springs, E_int, recursion inputs (step 3) */
#define PIMD_PROF_CHAIN 2     /* forward + backward recursions with the panel workers' force sums (steps 4, 5), and, as the
                                 tail of the same launch, the near-diagonal force band, Eq. 13 and the exterior forces (step 6) */
#define PIMD_PROF_ASSEMBLE 3  /* step 6 for xi = 0 (every ring closes on itself) */
#define PIMD_PROF_FINALIZE 4  /* V_B, sign, <E_c>; estimator arithmetic */
#define PIMD_PROF_INTEGRATE 5 /* velocity Verlet + thermostat (step 7) */
#define PIMD_PROF_COMBINE 6   /* force output */
#define PIMD_PROF_PAIR 7      /* pair forces (step 2) */
#define PIMD_PROF_EMAT 8      /* pimd_cycle_energies: the N x N write */
#define PIMD_PROF_PRMAT 9     /* pimd_connection_probabilities: the N x N write */
#define PIMD_PROF_GR 10       /* pair-distance histogram (estimator steps, pimd_set_pair_histogram) */
#define PIMD_PROF_SHARD 11    /* bead shards: boundary pack / E_int assembly */
#define PIMD_PROF_NSLOTS 12
/* mode 0: off.  PIMD_PROFILE_EVENTS: event pairs only -- the kernels run exactly as in a production step, so these are
 * the per-kernel times to quote.  PIMD_PROFILE_PHASES: also arms the clock64 phase counters inside the chain CTA
 * (pimd_get_chain_phases); the instrumented recursion kernel runs a few per cent slower, so its event time is an upper
 * bound in this mode.  Either mode turns graph replay off (every kernel is launched individually). */
#define PIMD_PROFILE_EVENTS 1
#define PIMD_PROFILE_PHASES 2
int pimd_set_profiling(pimd_t h, int mode);
int pimd_get_profile(pimd_t h, double *ms_host, uint64_t *count_host);
/* Phase clock of the recursion (steps 4, 5).  In profiling mode PIMD_PROFILE_PHASES the forward chain CTA adds up SM
 * cycles per phase of its 32-row blocks (HOST out, 16 entries, accumulated since the previous call, then reset).
 * Evaluations that ran with the previous evaluation's gauge (k_chain_spec: every evaluation of a handle but its
 * first) fill
 *   [0] wait at the block barrier (the helper warps or the workers' panel are late), [1] the dependent warp's
 *   prologue, [2] its 32 dependent steps (DFMA + SHFL), [3] its epilogue; measured from the barrier, one warp each:
 *   [4] a helper warp has its share of the next M tile, [5] of the older column blocks too, [8] of everything
 *   ([13], [14]: two more helper warps, on the other scheduler partitions), [7] the last block's columns are published,
 *   [9] the workers' panel is fetched ([10]: reads of the panel words it took, one per block = it never waited),
 *   [15] gauges, exponent tables and prefetch of the blocks ahead are in place; counts, not cycles: [11] batches of
 *   exponentials the helper warps met (older column blocks, E' tiles), [12] how many of them were skipped because every
 *   entry lay below e^-260 of its row's gauge, [6] blocks whose exponent arguments were formed in the factorised way.
 * Evaluations with a fresh max-plus gauge (k_chain) fill [0] loop overhead, [2k-1] the dependent warp's own time
 * in phase k = 1..4 (1 max-plus pass, 2 exponentials, 3 linear pass, 4 publish), [2k] its barrier wait. */
int pimd_get_chain_phases(pimd_t h, uint64_t *cycles_host);

/* Measured FP64 FMA issue rate of the device (a register-resident DFMA loop over all SMs; used
 * as the ALU roofline denominator).  tflops is HOST out (2 flop per DFMA). */
int pimd_probe_fp64_peak(void *cuda_stream, double *tflops);

/* The device exponentials of the hot kernels, element-wise, for accuracy tests: y[i] = f(x[i]) with
 * which = 0: exp_fast(x) (x <= 700), 1: exp_tab(x) (table of 32, x <= 700), 2: exp_neg_tab64(x) = exp(-x), x >= 0
 * (the recursion's and the force pass's table exponential; returns e^-708 for x > 708), 3: exp_neg_tab256(x) = exp(-x),
 * x >= 0 (the pair kernel's Gaussian, table of 256; returns e^-708 for x > 708).  x_dev, y_dev DEVICE, n elements.
 * Synchronises. */
int pimd_selftest_exp(void *cuda_stream, int which, const double *x_dev, double *y_dev, size_t n);

const char *pimd_last_error(pimd_t h); /* h may be NULL: error of the last failed pimd_create */
const char *pimd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PIMD_H */
