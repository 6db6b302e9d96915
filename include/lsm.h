/* lsm.h -- C ABI of the B200-native lattice-spring-model (LSM) step library, liblsm_b200.so.
 *
 * What it is: the hot path of CuLSM (arXiv 2201.04565, "ImageMech"): one time step of a bonded particle-spring
 * network, parallelised over the spring list, i.e.
 *   (1) truncated-harmonic spring forces  F_i = -sum_j k (r_ij - r0_ij) (r_i - r_j)/|r_i - r_j|   (Eq. 2)
 *   (2) the irreversible breakage test    r_ij > r_c  => the spring is dead for good
 *   (3) velocity Verlet in half-step-velocity form with fixed / displacement-controlled boundary rows
 *                                                                                    (Eq. 3-5)
 *   (4) device-side reductions: boundary reaction force, elastic energy U (Eq. 1), kinetic energy,
 *       broken-spring count (the paper sums U and KE on the CPU, and names "parallel reduction" as
 *       future work, L198).
 * Everything between lsm_create and lsm_read_* runs in hand-written CUDA kernels for sm_100a.  There is no CPU
 * fallback: without a CUDA device every compute entry point returns LSM_E_CUDA.
 *
 * Conventions
 *   - plain C; no exceptions or C++ types cross the boundary; every function returns lsm_status unless noted.
 *   - dim = 2 is the tuned path (all configurations of the paper and of BASELINE.json are 2-D).  dim = 3 (the layout of
 *     the paper's kernel listing) has the same semantics and entry points, vectors [N*3], on the
 *     streamed kernel with 32-byte records (or the plain direct kernel); no scatter path there.
 *   - HOST pointers unless a parameter says DEVICE.  Vector arrays are interleaved [N*dim] (x0 y0 x1 y1 ...) as in the
 *     paper's flattened 1-D arrays.  Inputs are borrowed for the duration of the call and copied;
 *     outputs are caller-allocated buffers of the documented size.  The handle owns all device memory.
 *   - particle ids / spring ids seen by the caller are ALWAYS the caller's own numbering, whatever renumbering
 *     (`reorder`) or compaction the library applies internally.
 *   - lsm_step only enqueues work on `stream`; lsm_read_* and lsm_sync synchronise it.  Errors are sticky: after a
 *     failure every later call on the handle returns the same code; lsm_last_error gives the text.
 *   - one handle may be used by one host thread at a time.
 */
#ifndef LSM_B200_H
#define LSM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LSM_MAX_GROUPS 8
#define LSM_ABI_VERSION 5

typedef struct lsm_sim lsm_sim; /* opaque */

typedef enum {
    LSM_OK = 0,
    LSM_E_INVALID = -1,     /* null pointer, bad enum, n < 0, dt <= 0, gamma < 0, wrong struct_size               */
    LSM_E_RANGE = -2,       /* spring endpoint outside [0,N), i == j, spring crossing two specimens, bad group id  */
    LSM_E_NONFINITE = -3,   /* NaN/Inf in x, v, m, k, r0, rc; m <= 0; r0 <= 0; k < 0; rc <= 0                      */
    LSM_E_CUDA = -4,        /* CUDA runtime error, or no CUDA device                                               */
    LSM_E_NOMEM = -5,       /* host or device allocation failed                                                    */
    LSM_E_STATE = -6,       /* the simulation failed earlier (e.g. non-finite energy detected on the device)       */
    LSM_E_UNSUPPORTED = -7  /* exact arithmetic with the scatter kernel, degree > 255 in the gather layout, a dim = 3
                               request for the scatter path                            */
} lsm_status;

enum { LSM_FIXED = 0, LSM_MOVE = 1 };                      /* boundary group modes */
/* force accumulation.  GATHER (= AUTO): particle-centric, no atomics, deterministic -- the product path.  The three
 * SCATTER modes are spring-centric as in the paper and are kept as measured comparisons:
 * SCATTER = one fp64 RED per force component and endpoint (the paper's atomicAdd design); SCATTER_WARP = springs sorted
 * by lower endpoint, segmented shuffle reduction, one RED pair per particle per warp; SCATTER_TILE = a CTA owns 1024
 * particles, every spring is evaluated once into its own shared-memory slot, particles sum their slots, one RED pair
 * per particle plus the spills across tile borders.  Fast arithmetic only (exact = 1 needs GATHER), dim = 2 only. */
enum { LSM_FORCE_AUTO = 0, LSM_FORCE_SCATTER = 1, LSM_FORCE_GATHER = 2, LSM_FORCE_SCATTER_WARP = 3, LSM_FORCE_SCATTER_TILE = 4 };
enum { LSM_REORDER_NONE = 0, LSM_REORDER_MORTON = 1, LSM_REORDER_RCM = 2,
       LSM_REORDER_BLOCKED = 3 /* 2-D only: bins of ~32 x 8 particles in row-major order, row-major inside a bin, so that a
                                  tile of 256 consecutive ids is a compact patch and neighbour offsets stay small */ };
/* kernels of the gather path: DIRECT = one thread per particle reading global memory; STREAMED = persistent CTAs,
 * bulk-async-copy (TMA engine) staging of the tile streams through a shared-memory mbarrier pipeline */
enum { LSM_GATHER_AUTO = 0, LSM_GATHER_DIRECT = 1, LSM_GATHER_STREAMED = 2 };
/* plain time steps of the streamed kernel: AUTO / ON = the producer also stages the tile's neighbour id ranges (its
 * "window": <= 4 contiguous ranges with a banded numbering) and the consumers gather from shared memory; OFF = gathers
 * from global memory (L1 / L2).  ON fails with LSM_E_UNSUPPORTED where AUTO would fall back to OFF. */
enum { LSM_WINDOW_AUTO = 0, LSM_WINDOW_ON = 1, LSM_WINDOW_OFF = 2 };
/* several time steps per launch: ON = one cooperative launch with a grid barrier between steps (state stays in L2 /
 * the CTAs' pipeline stages); RESIDENT = one thread-block cluster per specimen keeps it in shared memory for the whole
 * run of steps, ghosts pushed through distributed shared memory onto the receiver's transaction barrier (needs dim = 2,
 * 16-bit neighbour offsets, specimens starting on multiples of 32 particles and fitting one cluster; else
 * LSM_E_UNSUPPORTED); AUTO = RESIDENT where the clusters fill the GPU or the lattice is tiny, else ON for L2-resident
 * launch-bound problems (up to 2^18 particles), else one launch per step.  gather_window = AUTO also applies only up to
 * 2^25 particles (above, the bulk-copied neighbour ranges miss L2: DESIGN.md). */
enum { LSM_FUSION_AUTO = 0, LSM_FUSION_ON = 1, LSM_FUSION_OFF = 2, LSM_FUSION_RESIDENT = 3 };

/* Optional device allocator (the Python binding passes PyTorch's caching allocator). */
typedef void *(*lsm_alloc_fn)(size_t bytes, void *user);  /* returns a DEVICE pointer, NULL on failure */
typedef void (*lsm_free_fn)(void *dptr, void *user);

typedef struct lsm_desc {
    uint32_t struct_size;             /* = sizeof(lsm_desc): ABI check                                           */
    int32_t dim;                      /* 2 or 3                                                                   */
    int64_t n_particles, n_springs;   /* N >= 1, M >= 0, both < 2^31 - 1                                          */
    int32_t n_batch;                  /* B >= 1 independent specimens stored as one disjoint union                */
    int32_t _pad0;
    const int64_t *particle_offsets;  /* [B+1] ascending, [0] = 0, [B] = N; NULL allowed when B == 1              */
    const int64_t *spring_offsets;    /* [B+1]; springs of specimen b are [off[b], off[b+1]) and join its own
                                         particles only                                                          */
    const double *x;                  /* [N*dim] initial positions                                                */
    const double *v;                  /* [N*dim] initial velocities, NULL = zeros                                 */
    const double *mass;               /* [N] or NULL -> mass_uniform ("particle masses ... by type") */
    double mass_uniform;
    const int32_t *spring_i, *spring_j; /* [M] endpoints, the paper's atom_i / atom_j          */
    const double *k, *r0, *rc;        /* [M] stiffness, rest length, breaking LENGTH (absolute, Table 1
                                         PAPER.md:L137-L141); a NULL pointer takes the *_uniform scalar          */
    double k_uniform, r0_uniform, rc_uniform;
    double dt, gamma;                 /* time step; viscous damping coefficient (force -gamma*v, Q7)    */
    int32_t sample_every;             /* record {step, R_g, U, KE, n_broken} when step % sample_every == 0; 0 off */
    int32_t history_capacity;         /* samples kept in the device ring (0 -> 1024); oldest overwritten          */
    int32_t compact_every;            /* drop dead springs from the device lists every this many steps; 0 never   */
    int32_t reorder;                  /* LSM_REORDER_*: internal particle renumbering for gather locality: Morton order of
                                         the initial positions, or reverse Cuthill-McKee on the spring graph        */
    int32_t force_mode;               /* LSM_FORCE_*: AUTO = GATHER                                               */
    int32_t exact;                    /* 1: IEEE sqrt/divide, no FMA contraction, each particle sums its springs in
                                         ascending caller spring id -> bit-identical to a serial loop over the
                                         spring list (GATHER only).  0: fast arithmetic (FMA, rsqrt)              */
    int32_t step_fusion;              /* LSM_FUSION_* (above)                                                     */
    int32_t gather_variant;           /* LSM_GATHER_*: AUTO = STREAMED when a tile's rows fit in shared memory    */
    int32_t gather_window;            /* LSM_WINDOW_*                                                             */
    int32_t device;                   /* CUDA device ordinal                                                      */
    int32_t _pad1;
    int32_t cluster_size;             /* RESIDENT stepping: CTAs per cluster, 0 = chosen by the library, else 1, 2, 4, 8, 16 */
    void *stream;                     /* cudaStream_t, NULL = the default stream                                  */
    lsm_alloc_fn alloc;               /* NULL -> cudaMalloc / cudaFree                                            */
    lsm_free_fn free_;
    void *alloc_user;
} lsm_desc;

/* Layout / traffic facts about a handle (for benchmarks and tests). */
typedef struct lsm_info {
    int64_t n_particles, n_springs;
    int64_t n_half_edges_stored;      /* gather: ELL slots incl. padding; scatter: list length                    */
    int64_t bytes_per_half_edge;      /* id (2 B offset, or 4 B when an offset does not fit) + parameter bytes per slot */
    int32_t param_mode;               /* 0 uniform, 1 typed (1 B), 2 k,r0 uniform + rc per spring, 3 k,r0 typed + rc per
                                         spring, 4 k, r0, rc all per spring.  Gather layout: a per-spring rc costs 1 B
                                         per half-edge (a conservative 8-bit filter on r^2; the exact fp64 rc is
                                         read only when r is close to it, so the decision is always the fp64 one)  */
    int32_t n_types;
    int32_t force_mode, exact, reorder, n_batch;
    int64_t device_bytes;             /* device memory owned by the handle                                        */
    int64_t kernels_launched;         /* cumulative count of kernels this handle enqueued                         */
    int64_t current_step;
    int32_t gather_variant;           /* resolved LSM_GATHER_* (0 for the scatter path)                           */
    int32_t pipeline_stages;          /* streamed variant: stages of the shared-memory pipeline                   */
    int64_t stage_bytes;              /* streamed variant: bytes per stage                                        */
    int32_t step_fusion;              /* 0: one launch per step; 1: cooperative multi-step launches; 2: cluster-resident */
    int32_t cluster_size;             /* cluster-resident stepping: CTAs per cluster (0 otherwise)                */
    int64_t resident_smem_bytes;      /* cluster-resident stepping: dynamic shared memory per CTA                 */
    int32_t window_particles;         /* windowed gathers: largest tile window in particles (0 = gathers from global memory) */
    int32_t window_stages;            /* windowed gathers: pipeline stages                                        */
} lsm_info;

/* Build a simulation from particle / spring arrays.  Copies everything (the caller may free its inputs afterwards),
 * validates, renumbers, builds the device layout, evaluates forces once at step 0 (so f, U are defined and a spring
 * already longer than rc is broken at step 0).  On failure *out = NULL and lsm_last_error(NULL) has the reason. */
lsm_status lsm_create(const lsm_desc *desc, lsm_sim **out);

/* Define boundary group `group` in [0, LSM_MAX_GROUPS): its particles become kinematic from now on
 * (never integrated; position = position at this call + (steps since this call) * disp_per_step; FIXED ignores
 * disp_per_step).  particle_ids: [n] caller numbering; a particle may be in at most one group.  Calling it again for
 * the same group releases the old members first.  ("boundary displacements are first applied".) */
lsm_status lsm_set_boundary(lsm_sim *sim, int32_t group, const int32_t *particle_ids, int64_t n, int32_t mode,
                            const double *disp_per_step /* [dim] */);

/* Advance n_steps time steps: velocity Verlet, Eq. 3-5 in half-step-velocity form (L76): boundary
 * displacement first (L88), kick - drift - spring forces (Eq. 2) with the breakage test (L98) - damping - kick;
 * samples every sample_every steps, compaction every compact_every.  Only enqueues work on `stream` (asynchronous);
 * n_steps < 0 -> LSM_E_INVALID; a launch failure is sticky (LSM_E_CUDA). */
lsm_status lsm_step(lsm_sim *sim, int64_t n_steps);

/* Overwrite positions and velocities (restart / perturbation) from HOST arrays [N*dim] in caller numbering; forces are
 * re-evaluated at the current step and kinematic particles take the new position as their origin.  v NULL = zeros. */
lsm_status lsm_write_state(lsm_sim *sim, const double *x, const double *v);

/* Positions and velocities of the completed state (what Eq. 3-5 hold after the last step) into caller-allocated HOST
 * arrays, caller numbering; a kinematic particle reports v = disp_per_step / dt.  Synchronises the stream; returns
 * LSM_E_STATE (sticky) if a non-finite energy was detected on the device. */
lsm_status lsm_read_state(lsm_sim *sim, double *x /* [N*dim] or NULL */, double *v /* [N*dim] or NULL */);
/* Spring force on every particle at the current positions, Eq. 2 (no damping term). */
lsm_status lsm_read_forces(lsm_sim *sim, double *f /* [N*dim] */);
/* Per-particle virial stress of the current state, Eq. 7 without the 1/Omega factor (the caller divides
 * by a volume): S[p] = {S_xx, S_yy, S_xy} = 1/2 sum_l (x^l - x^p) (x) f^pl - m v (x) v, tension positive; broken
 * springs contribute nothing.  dim = 3: S[p] = {S_xx, S_yy, S_zz, S_xy, S_yz, S_zx}.  Gather layout only
 * (LSM_E_UNSUPPORTED with force_mode = SCATTER). */
lsm_status lsm_read_virial(lsm_sim *sim, double *S /* [N*3], dim = 3: [N*6] */);
/* Per-particle Lagrangian strain of the current state, Eq. 8 (eps^L = (J J^T - delta)/2, printed with its
 * summation lost; L156: "J is the locally affine transformation matrix considering the relative displacement of particle
 * with its first nearest neighbors"; reading Q21 of DESIGN.md).  For particle p, F = (sum d (x) d0)(sum d0 (x) d0)^-1 is the
 * least-squares affine map of the reference bond vectors d0 = xref_l - xref_p of its springs that are ALIVE now onto
 * their current bond vectors d = x_l - x_p; xref = the positions given to lsm_create (lsm_write_state does not move the
 * reference); E[p] = (F^T F - I)/2 = {e_xx, e_yy, e_xy}, dim = 3: {e_xx, e_yy, e_zz, e_xy, e_yz, e_zx} (symmetric;
 * tensor components, not engineering shear).  ok[p] (may be NULL) = 0 where p has fewer than dim independent live bonds
 * (det V <= 1e-12 (tr V / dim)^dim): E[p] = 0 there, never NaN.  Caller numbering; gather layout only (LSM_E_UNSUPPORTED
 * with a SCATTER force_mode).  The first call uploads the reference positions (16 or 32 bytes per particle of device
 * memory from then on).  Synchronises the stream. */
lsm_status lsm_read_strain(lsm_sim *sim, double *E /* [N*3], dim = 3: [N*6] */, uint8_t *ok /* [N] or NULL */);
/* Irreversible breakage, caller spring numbering: broken[s] = 1 if spring s is dead;
 * break_step[s] = step of the force evaluation that broke it, -1 if alive; *n_broken = total over all specimens. */
lsm_status lsm_read_broken(lsm_sim *sim, uint8_t *broken /* [M] or NULL */, int64_t *break_step /* [M] or NULL */,
                           int64_t *n_broken /* scalar or NULL */);
/* Per-specimen energies of the current state: U = sum over alive springs of k (r - r0)^2 / 2 (Eq. 1) and
 * KE of the free particles (PAPER.md:L113 sums them on the CPU; here a deterministic device reduction). */
lsm_status lsm_read_energy(lsm_sim *sim, double *U /* [B] or NULL */, double *KE /* [B] or NULL */);
/* Copy out (and clear) the samples recorded since the last call, oldest first, at most `capacity`:
 * step[n], reaction[n][B][LSM_MAX_GROUPS][dim] (raw sums of spring forces over each group's particles; the caller
 * divides by a cross-section to get stress), U[n][B], KE[n][B], n_broken[n][B] (cumulative).  NULL outputs skipped. */
lsm_status lsm_read_stress(lsm_sim *sim, int64_t capacity, int64_t *n_samples, int64_t *step, double *reaction,
                           double *U, double *KE, int64_t *n_broken);

/* Quasi-static driver for the paper's fracture protocol ("termination check each step", L143 grips
 * displaced apart): advance in chunks that end on sample steps until, for EVERY specimen, the reaction |R[group][axis]|
 * has fallen below stop_fraction (in [0,1)) of that specimen's own running peak (Q20), or max_steps have been
 * taken.  Needs sample_every > 0.  steps_done: steps taken by this call; failed: 1 if the criterion fired;
 * peak[B], peak_step[B]: the peak reaction magnitude seen during this call and its step (any may be NULL).  The samples
 * stay in the history ring for lsm_read_stress (the ring keeps the newest history_capacity of them). */
lsm_status lsm_run_to_failure(lsm_sim *sim, int64_t max_steps, int32_t group, int32_t axis, double stop_fraction,
                              int64_t *steps_done, int32_t *failed, double *peak, int64_t *peak_step);

/* Strain-rate control of the paper's protocol ("boundary particles were displaced apart ... at the strain
 * rate of 1e-6"): groups group_lo and group_hi (both already defined with lsm_set_boundary) become MOVE groups pulled
 * apart along `axis` so that the gauge length H0 -- the distance between the two groups' mean positions along the axis
 * at this call -- grows by strain_per_step * H0 per step: symmetric != 0 moves group_lo by -du/2 and group_hi by +du/2
 * per step (both grips, as in the paper), symmetric == 0 holds group_lo and moves group_hi by du.  ramp != 0 also gives
 * every free particle, along the axis, the velocity e (x - c) / dt of the affine field (c = the point that stays at rest)
 * so that the pull starts without a grip shock, and refreshes the held forces as lsm_write_state does.  *gauge_length
 * (may be NULL) returns H0: strain after n steps = n * strain_per_step.  dim = 2.  Synchronises the stream. */
lsm_status lsm_set_strain_rate(lsm_sim *sim, int32_t group_lo, int32_t group_hi, int32_t axis, double strain_per_step,
                               int32_t symmetric, int32_t ramp, double *gauge_length);

/* Drop dead springs from the device lists now (also done every compact_every steps; the paper keeps dead springs with
 * k = 0, L196).  Two stages, both on the device and asynchronous: every row is compacted in place, stably (each particle
 * keeps its summation order, so no result changes); then the slot storage is repacked (prefix sum of the slices' live
 * widths, stable move) so that the streams the step kernel copies shrink.  A slice of 32 particles stores as many slots
 * per particle as its longest row: bytes fall only where every row of a slice lost springs. */
lsm_status lsm_compact(lsm_sim *sim);
lsm_status lsm_sync(lsm_sim *sim);                                   /* cudaStreamSynchronize on the handle's stream */
lsm_status lsm_get_info(lsm_sim *sim, lsm_info *info);               /* never fails on a valid handle, even after an error;
                                                                         synchronises the stream once after a compaction (slot count) */
/* Device pointers of the current state in INTERNAL numbering, for zero-copy consumers (may change after lsm_step):
 * records of 2 doubles {x, y} per particle for dim = 2, of 4 doubles {x, y, z, 0} for dim = 3; owned by the handle. */
lsm_status lsm_device_state(lsm_sim *sim, const double **pos_xy /* DEVICE */, const double **vel_xy /* DEVICE */);
const char *lsm_last_error(const lsm_sim *sim); /* sim NULL: error of the last failed lsm_create on this thread */
void lsm_destroy(lsm_sim *sim);
int32_t lsm_abi_version(void);

/* ---- The one entry point that allocates nothing ----------------------------------------------------------------------
 * Elastic energy U = sum over unbroken springs of k (r - r0)^2 / 2 (Eq. 1; the quantity of Fig. 4B, which
 * the paper sums on the CPU, L113) of a spring list the caller already holds ON THE DEVICE, without an lsm_sim handle.
 *
 * Why it exists: every other call needs a handle, and lsm_create makes dozens of device allocations.  This one is for
 * callers that cannot ask CUDA for memory at the point where they need the number: a process whose GPU memory was all
 * given to one arena or framework pool at start-up (cudaMalloc fails there, or eats what the pool's owner budgeted); a
 * monitor running beside asynchronous lsm_step work (cudaFree waits for the whole device and cudaMalloc may, which stalls
 * the step pipeline); a long unattended sweep whose memory footprint must be fixed when the library loads.  The function
 * calls neither cudaMalloc nor cudaFree nor any allocating library routine.  Its only scratch -- the per-block partial
 * sums of a deterministic two-level reduction -- lives in a fixed array inside the library: 524,544 bytes that every GPU
 * which loads liblsm_b200.so holds until the process exits, whether or not this function is ever called.
 *
 * The limit: n_springs <= LSM_STATIC_MAX_SPRINGS (2^28; one partial per 8192 springs, 32768 partials).  A longer list is
 * rejected with LSM_E_RANGE before anything is enqueued and U is left untouched: split the list and add the parts, or
 * use lsm_create + lsm_read_energy.
 *
 * Arguments (DEVICE pointers are memory of `device`, in the CALLER's numbering; nothing is copied or kept):
 *   device, stream   CUDA device ordinal (made current for the call, the caller's device restored) and cudaStream_t
 *                    (NULL = default stream).  The call only enqueues a 8-byte memset and two kernels on `stream`.
 *   dim              2 or 3; x is interleaved [n_particles*dim] as everywhere in this header.
 *   spring_i/j       [n_springs] endpoints (the paper's atom_i / atom_j, L91-L92); may be NULL when n_springs == 0.
 *   k, r0            [n_springs], or NULL to take k_uniform / r0_uniform.
 *   broken           [n_springs] bytes, non-zero = the spring is dead and contributes nothing (what lsm_read_broken
 *                    returns, uploaded); NULL = all alive.  Breakage is irreversible (L98, L196): this function does not
 *                    test r > rc itself, the flags are the caller's record of it.
 *   U                DEVICE [1]: the energy.  Summation order is fixed by the list alone (same bits on every GPU).
 *   counts           DEVICE [2] or NULL: {springs summed, springs skipped because an endpoint is outside
 *                    [0, n_particles) or i == j}.  Bad ids are skipped and counted on the device, never dereferenced.
 *   errbuf           HOST buffer of errbuf_len bytes for the message of a failed call (may be NULL); lsm_last_error
 *                    does not cover this function.
 * Returns LSM_OK once the work is enqueued (read U after synchronising the stream); LSM_E_INVALID (bad dim / sizes /
 * NULL pointers / device ordinal outside [0, 64)), LSM_E_RANGE (list too long), LSM_E_CUDA (no device, launch failure).
 *
 * Sharing: all calls on one device use the same array, and it keeps whatever the previous call left in it.  The function
 * clears the one word that must start at zero (the bad-id counter) itself, on `stream`, and every partial it reads was
 * written by the same call, so calls that follow each other on one stream, or that are otherwise ordered, are
 * independent of each other.  Two calls that may run on the GPU at the same time (different streams or host threads
 * without an event or synchronisation between them) race on the array and both results are garbage: order them.
 *
 * First call on each device: looks up the device address of the array (cudaGetSymbolAddress, once per device, under a
 * host mutex).  Make that first call on an ordinary stream, before any stream capture is begun. */
#define LSM_STATIC_MAX_SPRINGS 268435456
lsm_status lsm_spring_energy_static(int32_t device, void *stream, int32_t dim, int64_t n_particles, int64_t n_springs,
                                    const double *x /* DEVICE */, const int32_t *spring_i /* DEVICE */, const int32_t *spring_j /* DEVICE */,
                                    const double *k /* DEVICE or NULL */, const double *r0 /* DEVICE or NULL */,
                                    double k_uniform, double r0_uniform, const uint8_t *broken /* DEVICE or NULL */,
                                    double *U /* DEVICE [1] */, int64_t *counts /* DEVICE [2] or NULL */,
                                    char *errbuf /* HOST */, size_t errbuf_len);

#ifdef __cplusplus
}
#endif
#endif /* LSM_B200_H */
