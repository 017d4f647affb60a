/*
 * mdpd.h -- C-ABI of the B200-native mDPD timestep library (libmdpd_b200.so).
 *
 * One full velocity-Verlet timestep of many-body dissipative particle dynamics for fluid and frozen
 * wall particles on ONE GPU (sm_100a), as stated in arxiv/paper_1903_10134:
 *   - pair forces F = F^R + F^D + F^C, weight functions, fluctuation-dissipation   PAPER.md L75   (sec. 2.1)
 *   - mDPD conservative force, Eq. (1), and the many-body density rho_i
 *   - velocity-Verlet order x -> rho -> f -> v                                      PAPER.md L125-133 (Algorithm 1)
 *   - body-force driving, dt = 0.01                                                 PAPER.md L186  (sec. 5.1)
 *   - frozen ("fixed") solid wall particles                                         PAPER.md L162  (sec. 4.2)
 * and the readings R1..R18 of DESIGN.md section 3 where the paper is silent (random-force 1/sqrt(dt), the pair
 * hash, bounce-back at a voxel mask, ...).
 *
 * Conventions
 *   - Every function returns int: MDPD_OK (0) or a negative error code.  Nothing throws, nothing exits.
 *     mdpd_last_error(h) returns a NUL-terminated description owned by the handle.
 *   - "host or device" pointers: any pointer cudaMemcpy(..., cudaMemcpyDefault) accepts.  The library copies; the
 *     caller keeps ownership of everything it passes in.
 *   - All device work is enqueued on the stream given to mdpd_create (0 = legacy default stream).
 *   - A handle is not thread-safe.  One handle = one simulation on one device.
 *   - There is no CPU fallback: without a CUDA device mdpd_create fails with MDPD_ECUDA.
 */
#ifndef MDPD_H_
#define MDPD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MDPD_OK 0
#define MDPD_EINVAL (-1)    /* bad argument / unsupported parameter value                         */
#define MDPD_ENOMEM (-2)    /* workspace too small or allocation failed                           */
#define MDPD_ECUDA (-3)     /* a CUDA runtime call failed (text in mdpd_last_error)               */
#define MDPD_EOVERFLOW (-4) /* neighbour-list capacity exceeded: raise mdpd_params.max_neigh      */
#define MDPD_ESTATE (-5)    /* call order (e.g. step before load_particles)                       */
#define MDPD_ENAN (-6)      /* a non-finite coordinate appeared                                   */
#define MDPD_EINSOLID (-7)  /* fluid particle(s) start inside a solid voxel                       */

typedef struct mdpd_ctx mdpd_ctx; /* opaque */

/* Plain-old-data; copied by mdpd_set_params.  Units: rc = 1, mass = 1, kT = 1 (DPD units). */
typedef struct {
  float box[3];           /* periodic box [0,Lx) x [0,Ly) x [0,Lz); each L >= 3 (rc + skin)                           */
  float rc, rd;           /* force and density cut-offs, rd <= rc (1.0, 0.75)      */
  float A, B;             /* Eq. (1): attractive A < 0, many-body repulsive B > 0 (-40, 25)   */
  float gamma, sigma;     /* dissipative / random amplitudes, sigma^2 = 2 gamma kT (4.5, 3.0)           */
  float kT;               /* informational: if > 0 the library checks |sigma^2 - 2 gamma kT| <= 1e-3 sigma^2          */
  float s;                /* exponent of wR = (1 - r/rc)^s, wD = wR^2, 0 < s <= 4 (1: the paper's) PAPER.md L75 (R15)  */
  float mass, dt;         /* particle mass (1), timestep (0.01)         */
  float g[3];             /* body acceleration on fluid particles         */
  float skin;             /* Verlet-list skin (default 0.25); list radius = rc + skin; rebuild when the largest
                             displacement since the last build exceeds skin/2                   DESIGN.md R3, R4      */
  float headroom;         /* capacity of a tile of cells (shared memory) = headroom x the fullest tile of the loaded
                             state; 0 = default: 1.15, lowered to no less than 1.08 where that keeps two CTAs of the force pass per SM.  Raise it when the density will grow locally during the run (a
                             contracting slab, a filling pore): outgrowing the capacity is MDPD_EOVERFLOW              */
  uint32_t seed;          /* seed of the pair hash      */
  uint32_t max_neigh;     /* list capacity per particle, <= 128; 0 = automatic                                       */
  uint32_t reorder_every; /* RESERVED, must be 0 or 1.  The list stores indices into the sorted tile image, so the sort
                             into Morton-ordered tiles cannot be skipped at a rebuild: it IS the reorder (R16) */
  uint32_t flags;         /* MDPD_FLAG_* */
} mdpd_params;

#define MDPD_FLAG_NO_GRAPH 1u /* launch kernels one by one instead of replaying the captured CUDA graph */
#define MDPD_FLAG_DIRECT 2u   /* list-free path: no Verlet list; every step finds the r < rc neighbours straight from the
                                 cells (same results; the cells are still re-sorted on the skin/2 displacement trigger).
                                 Fixed by mdpd_load_particles. */
#define MDPD_FLAG_TMA_STAGING 4u     /* BOTH tile passes stage their tile with cp.async.bulk (1-D TMA bulk copies, one per */
#define MDPD_FLAG_CPASYNC_STAGING 8u /* contiguous run, mbarrier completion) / with per-particle cp.async copies.  Default
                                        (neither flag): bulk copies in the density pass, cp.async in the force pass, as
                                        measured in profiles/r2_staging.md.  Same results either way.  Fixed by load. */

/* Create a handle on CUDA device `device`; `cuda_stream` is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream)
 * or NULL for the default stream.  The handle must be destroyed with mdpd_destroy. */
int mdpd_create(mdpd_ctx** out, int device, void* cuda_stream);
int mdpd_destroy(mdpd_ctx* h);

/* Validate and store parameters.  Before load_particles: any field.  After load_particles only g, dt, seed, A, B,
 * gamma, sigma, kT may change (box, cut-offs, skin, capacities are frozen: MDPD_ESTATE otherwise). */
int mdpd_set_params(mdpd_ctx* h, const mdpd_params* p);

/* Per-type-pair conservative parameters of Eq. (1) ("the particle interaction force between two types
 * of materials such as solid and liquid can be modified by adjusting A_SL, B_SL"; Tables 1 and 2, PAPER.md L155-160,
 * L188-192; five material types in the kerogen case, L247).  A, B: [ntypes][ntypes] float32 row-major HOST arrays,
 * symmetric (else MDPD_EINVAL), ntypes <= 8.  After this call the `type` byte of mdpd_load_particles is the SPECIES
 * index s in [0, ntypes) (a larger value: MDPD_EINVAL at load), the pair (i, j) uses A[s_i][s_j], B[s_i][s_j] in place
 * of mdpd_params.A / .B, and species s is frozen (never integrated, v = 0, R8) iff bit s of frozen_mask is
 * set.  rc, rd stay those of mdpd_params for every pair; gamma, sigma too unless mdpd_set_pair_gamma_sigma is used.  Call before mdpd_load_particles; afterwards
 * only the VALUES may change (same ntypes and frozen_mask, else MDPD_ESTATE).  ntypes = 0 returns to one material
 * (type byte != 0 <=> frozen wall). */
int mdpd_set_pair_params(mdpd_ctx* h, uint32_t ntypes, const float* A, const float* B, uint32_t frozen_mask);

/* Per-type-pair dissipative and random amplitudes (every pair carries F^D = -gamma w_D (e.v) e and
 * F^R = sigma w_R xi e with sigma^2 = 2 gamma kT; the paper runs water at gamma = 12.4, L141, and its other fluids at 4.5,
 * L89 and L186, so a run with two fluids needs them per pair of species).  gamma, sigma: [ntypes][ntypes] float32
 * row-major HOST arrays, symmetric, >= 0 (else MDPD_EINVAL); ntypes must be that of the preceding mdpd_set_pair_params
 * (else MDPD_EINVAL).  The pair (i, j) then uses gamma[s_i][s_j], sigma[s_i][s_j] in place of mdpd_params.gamma / .sigma.
 * Nothing is checked against kT: sigma_ij^2 = 2 gamma_ij kT is the caller's choice.  NULL for either matrix returns to the
 * uniform amplitudes; so does a later mdpd_set_pair_params with another ntypes.  May be called before or after
 * mdpd_load_particles (new values enter the next force evaluation).  The paper also names a per-pair r_d (L153); it is
 * NOT offered: r_d = 0.75 r_c "for all particle interactions" (L81, L89) and a per-pair r_d would change the density
 * weight itself (R22). */
int mdpd_set_pair_gamma_sigma(mdpd_ctx* h, uint32_t ntypes, const float* gamma, const float* sigma);

/* Device bytes needed for n particles (+ an optional mask of mask_dims = {nx, ny, nz} voxels).  Returns 0 on bad input. */
size_t mdpd_workspace_bytes(const mdpd_params* p, uint64_t n, int has_mask, const uint32_t mask_dims[3]);

/* Give the library its device memory: `dev_ptr` (256-byte aligned, >= mdpd_workspace_bytes) is OWNED BY THE CALLER
 * (e.g. a torch uint8 tensor) and must outlive the handle (or the next mdpd_set_workspace).  If never called,
 * load_particles allocates with cudaMalloc (and re-allocates when a later load needs more) and mdpd_destroy frees that
 * allocation.  Calling it on a handle that already holds particles drops them: the next call must be
 * mdpd_load_particles.  With a caller-owned workspace the stepping path (load, step, get_state, compute_forces,
 * compute_virial, counters) never allocates device memory; the two diagnostics mdpd_get_pairs and mdpd_rng_fill are
 * the exception (see there). */
int mdpd_set_workspace(mdpd_ctx* h, void* dev_ptr, size_t bytes);

/* Load n < 2^28 particles.  pos, vel: [n][3] float32, host or device.  type: [n] uint8 (0 = fluid, any other value =
 * frozen wall; after mdpd_set_pair_params: the species index) or NULL (all fluid / species 0).  The tag of a particle is
 * its index in this call and is permanent.  Positions are wrapped into the box;
 * frozen particles get v = 0.  Builds the cell list / neighbour list and evaluates rho and f at step index 0.
 * n = 0 is allowed.  Synchronises the stream. */
int mdpd_load_particles(mdpd_ctx* h, uint64_t n, const float* pos, const float* vel, const uint8_t* type);

/* Optional voxel mask for the no-slip bounce-back (R7): mask[nz][ny][nx] uint8, 1 = solid, host or device;
 * dims = {nx, ny, nz}; nx * voxel == Lx etc.  NULL clears the mask.  Call after load_particles (the workspace must have
 * been sized with the mask).  Returns MDPD_EINSOLID if a fluid particle lies in a solid voxel (count in last_error). */
int mdpd_load_wall_mask(mdpd_ctx* h, const uint8_t* mask, const uint32_t dims[3], float voxel);

/* Advance nsteps velocity-Verlet steps (Algorithm 1).  Asynchronous on the stream: device-side
 * faults (list overflow, NaN) are latched and reported by the next synchronising call (get_state, get_counters). */
int mdpd_step(mdpd_ctx* h, uint32_t nsteps);

/* Copy the state out in TAG order.  pos, vel, force: [n][3] float32; rho: [n] float32; any pointer may be NULL; host or
 * device.  vel are the full-step velocities; force and rho are those of the last force evaluation.  Forces on frozen
 * particles are reported only after mdpd_compute_forces (the step path does not compute them: they are never used).
 * Synchronises the stream and returns a latched device fault if there is one. */
int mdpd_get_state(mdpd_ctx* h, float* pos, float* vel, float* force, float* rho, uint64_t* step);

/* Checkpoint / resume.  A state is (pos, vel, force, step) as mdpd_get_state returns them: the force of time level k
 * was evaluated with the half-step velocities (Algorithm 1 order, R6), so it is part of the state and cannot
 * be recomputed from the full-step velocities.  Resume = mdpd_load_particles(pos, vel, type) +
 * mdpd_set_step_counter(step) + mdpd_set_forces(force).
 * mdpd_set_step_counter sets the step index used by the hash (forces are NOT recomputed).
 * mdpd_set_forces overwrites the stored forces; force: [n][3] float32 in TAG order, host or device. */
int mdpd_set_step_counter(mdpd_ctx* h, uint64_t step);
int mdpd_set_forces(mdpd_ctx* h, const float* force);

/* ---- parity / diagnostics exports (the GPU-vs-oracle comparison needs them) ---- */

/* rho and f (on every particle, frozen ones included) from the current x, v at the current step index.
 * NOTE: this REPLACES the stored force (and rho).  The force of a time level is part of the state (it was evaluated with
 * the half-step velocities, see the checkpoint note above), so a call made between two mdpd_step calls changes the first
 * half kick of the next step, i.e. the trajectory (by O(dt^2); the oracle's mdpd_ref_compute_forces has the same
 * semantics).  To look at forces without touching the run, save get_state's force first and give it back with
 * mdpd_set_forces.  The same holds for mdpd_compute_virial. */
int mdpd_compute_forces(mdpd_ctx* h);

/* mdpd_compute_forces, and in the same pass the configurational (conservative-force) part of the stress:
 * out = sum over interacting pairs of r_ij,a F^C_ij,b for ab = xx, yy, zz, xy, xz, yz (F^C of Eq. (1), PAPER.md L77-81;
 * frozen-frozen pairs excluded as in the force).  With the kinetic part sum m v_a v_b from mdpd_get_state this gives the
 * pressure tensor, and for a slab normal to x the interfacial tension of section 4.1. */
int mdpd_compute_virial(mdpd_ctx* h, double out[6]);

/* All tag pairs (a < b) with r < rcut, found through the Verlet list with the kernels' own fp32 predicate
 * (r^2 < rcut^2); rcut <= rc + skin.  For rcut > rc the result is complete only right after a list build
 * (load_particles, or any step that rebuilt).  *count receives the number found; up to cap pairs are written
 * to `pairs` ([cap][2] uint32, HOST memory), sorted lexicographically.
 * Diagnostic: allocates its scratch (8 bytes per pair of `cap`) with cudaMalloc and frees it before returning, also
 * when a workspace was given; not meant for the stepping loop.  On the list-free path (MDPD_FLAG_DIRECT) it first
 * builds a list from the current cells. */
int mdpd_get_pairs(mdpd_ctx* h, float rcut, uint64_t* count, uint32_t* pairs, uint64_t cap);

/* mdpd_get_pairs without any device allocation, for callers that cannot make one.
 *
 * Who that is: a host program that has already handed all free device memory to its own pool (a tensor framework's
 * caching allocator, a job that reserves the whole card at start-up) -- there a cudaMalloc from inside this library
 * simply fails with out-of-memory although the pool has room; and code on a latency-critical path shared with other
 * streams, because cudaMalloc / cudaFree make the whole device wait, not only this handle's stream.  mdpd_get_pairs
 * does two cudaMalloc + two cudaFree per call; this variant does none, and calls no other allocating runtime or
 * library routine.
 *
 * How: the scratch of the pair search (an 8-byte hit counter and the unsorted pair buffer) is a fixed array inside the
 * library image instead: 256 + 8 * MDPD_STATIC_PAIRS_MAX bytes (about 4 MiB) of every GPU that loads the library,
 * held until the process exits.  Arguments, result and errors are those of mdpd_get_pairs (same kernel, same fp32
 * predicate, same sorted output in HOST memory `pairs`; inputs and outputs stay the caller's), except:
 *   - cap > MDPD_STATIC_PAIRS_MAX is refused with MDPD_EINVAL (text in mdpd_last_error) before anything runs.  As in
 *     mdpd_get_pairs, *count may exceed cap: it is the number found, of which the first cap in device order are kept.
 *   - MDPD_ESTATE between mdpd_profile_begin and mdpd_profile_end (the per-kernel timing creates events on demand).
 *   - The handle's own workspace must already exist (mdpd_load_particles has run); with mdpd_set_workspace that one is
 *     the caller's memory too.
 *   - The first call on a device is also a set-up call: it looks up the array's device address
 *     (cudaGetSymbolAddress, once per device, return code checked).  Make that first call before any stream capture
 *     is begun on the device.
 *   - ONE array per device serves every handle and every call, and it keeps what the last call wrote.  The library
 *     zeroes the counter at the start of each call (on the handle's stream); the pair slots need no clearing.  Two
 *     calls whose GPU work can overlap -- two handles on different streams, two host threads -- race on the array
 *     and return garbage: serialise them yourself.  A handle is not thread-safe anyway.
 * Synchronises the handle's stream. */
#define MDPD_STATIC_PAIRS_MAX 524288u
int mdpd_get_pairs_static(mdpd_ctx* h, float rcut, uint64_t* count, uint32_t* pairs, uint64_t cap);

/* Run the DEVICE hash kernel: out[q] = HASH(min(pairs[q]), max(pairs[q]), step, seed of the handle).
 * pairs: [npairs][2] uint32, out: [npairs] uint32, host or device.  Diagnostic: allocates 12 bytes per pair with
 * cudaMalloc and frees them before returning. */
int mdpd_rng_fill(mdpd_ctx* h, uint64_t npairs, const uint32_t* pairs, uint32_t step, uint32_t* out);

#define MDPD_NCOUNTERS 16
/* out[0] steps done, [1] list rebuilds, [2] bounce-back events, [3] longest neighbour list at the last build,
 * [4] sum over particles of the list lengths at the last build, [5] most particles staged in shared memory by one
 * tile (tile + halo) at the last build, [6] device fault events (list / tile overflows + non-finite coordinates; also
 * latched as an error code), [7] kernels launched by this handle so far, [8] sum over all density passes so far of
 * the in-range (r < rc) neighbour counts = pair evaluations of the force passes, [9] number of density passes so far,
 * [10] tile shape tx | ty << 8 | tz << 16 (cells: the largest extent; tiles along a dimension differ by at most one cell),
 * [11] number of tiles; [12..15] reserved (0).
 * Synchronises the stream. */
int mdpd_get_counters(mdpd_ctx* h, uint64_t out[MDPD_NCOUNTERS]);

const char* mdpd_last_error(const mdpd_ctx* h);

/* ---- measurement: per-kernel device times of the step path (CUDA events on the handle's stream) ---- */
#define MDPD_PROF_SLOTS 16
/* Start bracketing every kernel this handle launches with a pair of CUDA events. */
int mdpd_profile_begin(mdpd_ctx* h);
/* Stop, synchronise the stream and return, per kernel slot, the summed device time [ms] and the launch count since
 * mdpd_profile_begin.  Slots past the last named one stay 0.  (Kernels of the rebuild chain are launched every step
 * and return at once when the displacement trigger did not fire: their launch count includes those.) */
int mdpd_profile_end(mdpd_ctx* h, double ms[MDPD_PROF_SLOTS], uint64_t launches[MDPD_PROF_SLOTS]);
/* Name of a kernel slot ("k_force", "k_density", ...; "" past the last one).  Static storage. */
const char* mdpd_profile_name(int slot);

/* The extra -D options this library was compiled with, sorted and comma-joined ("" for the plain build;
 * "-DMDPD_CHECKS" for the build with the kernels' own bounds checks, "-DMDPD_FIRST_TILE=..." for a measurement build).
 * bench.py prints it in its JSON line so that a timing can never be taken on a checks build unnoticed.  Static storage. */
const char* mdpd_build_flags(void);

/* Issue-rate probe for the ALU roofline: runs three short register-only kernels on `device`
 * (every SM, 64 resident warps, 8 independent dependency chains per thread), timed with CUDA events on `cuda_stream`, and
 * returns warp-instructions per second of the whole GPU: out[0] FP32 FMA (FFMA), out[1] logic pipe (LOP3 + VIMNMX),
 * out[2] 32 x 32 -> 64 integer multiply (IMAD.WIDE, the hash's multiply); out[3] = the SM clock [Hz] the runtime
 * reports as maximum.  No handle needed.  Returns MDPD_OK or MDPD_ECUDA. */
int mdpd_probe_issue_rates(int device, void* cuda_stream, double out[4]);


#ifdef __cplusplus
}
#endif
#endif /* MDPD_H_ */
