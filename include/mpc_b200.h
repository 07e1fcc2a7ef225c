/* mpc_b200.h -- C ABI of the B200-native multiparticle collision dynamics (MPC) fluid step.
 *
 * What one call of mpc_step(ctx, 1) computes (arXiv 2406.15236 "HTMPC", cited as PAPER.md:<line>):
 *   MOVE              r_i <- r_i + h v_i                          Eq. (1)
 *                     (+ constant acceleration; bounce-back at no-slip walls)
 *   PROCESS           random shift of the collision lattice, cell index of every particle,
 *                     per-cell sums (count, momentum, energy, ...)
 *   REORDER           every `rebin_every` steps the particles are re-sorted by (cell key, id)
 *                     (counting sort: histogram, prefix sum, scatter)
 *   PROCESS_CELLS     v_cm, rotation axis, thermostat factor kappa   Eqs. (2),(5)-(7)
 *   ROTATE_VELOCITIES v_i <- v_cm + kappa D(alpha)(v_i - v_cm) [+ omega x r_ic]   Eqs. (2)-(5)
 *                     or MPC-AT: v_i <- v_cm + v_ran_i - mean(v_ran) [+ omega x r_ic]  (U5)
 * in the paper's order (Fig. 1c). Random numbers are Philox-4x32-10 blocks with
 * key = seed and counter = (index, sub, step, tag); the stream layout is fixed in DESIGN.md "RNG".
 *
 * Conventions
 *   - Every function returns an int status: MPC_OK (0) or a negative MPC_E* code. Nothing throws,
 *     aborts or prints. mpc_last_error() gives a message for the last failure on that context.
 *   - "device pointer" = CUDA global memory of the current device; "host pointer" = ordinary host
 *     memory (pinned memory makes the *_host copies asynchronous to the host, nothing else changes).
 *   - The library never allocates device memory. The caller (e.g. a torch tensor) owns the
 *     workspace passed to mpc_bind and every buffer passed to set/get calls; the library owns only
 *     the host-side context, released by mpc_destroy.
 *   - All work is enqueued on the CUDA stream given to mpc_bind. Calls that return data to the host
 *     (mpc_observables, mpc_get_state_host) synchronise that stream; the others do not.
 *   - Particle arrays are fp32 structure-of-arrays x,y,z,vx,vy,vz plus a uint32 id per particle
 *     (PAPER.md:170). The internal particle order changes at every reorder; get_state returns the
 *     particles sorted by (memory key, id) as of the last reorder step, together with the ids (see
 *     mpc_get_state; the caller un-permutes by id).
 *   - Not thread-safe per context; different contexts are independent.
 */
#ifndef MPC_B200_H
#define MPC_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MPC_OK      0
#define MPC_EINVAL -1 /* bad argument or unsupported combination of options            */
#define MPC_ESTATE -2 /* call order: step before bind/set_state, get_cells before a step */
#define MPC_ENOMEM -3 /* workspace too small for the requested number of particles      */
#define MPC_ECUDA  -4 /* a CUDA call failed; sticky until mpc_destroy                   */
#define MPC_ERANGE -5 /* mpc_observables: velocities left the range of the fixed-point cell sums */

typedef struct mpc_ctx mpc_ctx; /* opaque */

typedef struct {
  int   collision;   /* 0 = SRD rotation (Eq. 2); 1 = MPC-AT (Andersen thermostat, U5)       */
  int   conserve_L;  /* 0 = -a; 1 = +a, cell-level angular-momentum conservation (Eqs. 3-4)            */
  int   thermostat;  /* 0 = none; 1 = cell-level Maxwell-Boltzmann scaling (Eqs. 5-7); ignored for AT  */
  float alpha;       /* SRD rotation angle in radians (cos/sin taken once in double, cast to fp32)     */
  float dt;          /* MPC time step h                                                                */
  float kT;          /* k_B T of the thermostat / of virtual wall particles / of MPC-AT                */
  float mass;        /* particle mass m (all fluid particles are identical)               */
  float g[3];        /* constant acceleration (force / mass); must be 0 along a wall normal            */
  int   bc[3];       /* per axis: 0 = periodic; 1 = no-slip walls at 0 and L: bounce-back v -> -v plus      */
                     /* virtual wall particles in wall-cut cells; 2 = slip walls: specular reflection, no  */
                     /* virtual particles (U7, U8, U20). At most one wall axis       */
  int   grid_shift;  /* 1 = random lattice shift in [-a/2,a/2)^3 every step; 0 = off     */
  int   rebin_every; /* reorder when step % rebin_every == 0; >= 1; MPC-AT requires 1                  */
  int   brick[3];    /* brick dims (powers of two <= 64) of the brick-major memory key; {1,1,1} = row-major.
                        Memory order only: results do not depend on it. {16,16,8} is the fast choice          */
  float shear_rate;  /* Lees-Edwards shear d v_x / d z (U21): the periodic images above /
                        below the box along z are displaced by +-shear_rate L_z t along x and move with
                        +-shear_rate L_z. 0 = off. Needs periodic boundaries on all axes, SRD without +a             */
  int   phantoms;    /* 1 = explicit phantom-particle set in the wall part of wall-cut cells (U22):
                        positions uniform in the wall part, velocities Gaussian about the wall velocity, number = wall
                        fraction x round(n_per_cell), rounded stochastically. Needs a no-slip wall axis and rebin_every = 1.
                        Required for +a and MPC-AT at walls. 0 = the velocity-only virtual particles of U8 (SRD -a only)  */
  unsigned solute_id0; /* embedded point-particle solutes (U23): particles with id >= solute_id0 */
  float solute_mass; /* ... have this mass instead of `mass` and take part in the collision with it (all cell sums are
                        mass-weighted; MPC-AT draws them from N(0, kT/solute_mass)). 0 = no solutes. Needs rebin_every = 1;
                        not with Lees-Edwards shear. Solutes stream ballistically like fluid particles                   */
  float wall_velocity; /* moving no-slip walls (plane Couette flow; U24): the wall at L moves with
                        +wall_velocity along x, the wall at 0 with -wall_velocity; bounce-back in the frame of the wall
                        (v -> 2 u_wall - v), wall / phantom particles thermal about u_wall. Needs bc = 1 on y or z            */
  int   sub_z0;      /* slab subdomain of a multi-GPU run: this context owns the cell layers    */
  int   sub_nz;      /* [sub_z0, sub_z0 + sub_nz) along z of the box given to mpc_create (the WHOLE box: cells[2] = all layers) and
                        holds one brick layer (brick[2] cell layers) of halo on either side. 0, 0 = the whole box (default).
                        Both multiples of brick[2]; sub_nz >= 2 brick[2]; sub_nz + 2 brick[2] <= cells[2]. Periodic SRD without +a,
                        walls, shear or force. The caller gives the rank the particles whose z lies in its layers; particles may
                        drift up to one brick layer outside (further: counted in n_range_overflows, results invalid); moving
                        them to the owning rank rides on the reorder (mpc_sub_begin) or is done with mpc_sub_pack.
                        See mpc_sub_connect, mpc_sub_begin, mpc_sub_end                                                        */
} mpc_params;

typedef struct {
  unsigned long long n;                /* number of particles                                          */
  double P[3];                         /* total momentum m * sum v                                     */
  double E_kin;                        /* (m/2) sum |v|^2                                              */
  double kT_est;                       /* m sum |v - <v>|^2 / (3 (N-1))                                */
  double kT_cell;                      /* sum_c m sum |v - v_cm,c|^2 / sum_c 3 (N_c - 1), cells with
                                          N_c >= 2, from the last step's pre-collision sums; 0 if none */
  unsigned max_cell_count;             /* largest N_c of the last step; 0 if no step was taken         */
  unsigned long long n_singular_cells; /* +a only: cells whose inertia tensor was rejected (U10)       */
  unsigned long long step;             /* step counter t                                               */
  unsigned long long n_range_overflows;/* events since the last mpc_set_state in which a value left the range the
                                          fixed-point cell sums are sized for ("overflows may occur ...
                                          invalidating the results"): a particle with |v| >= 8 u, u = sqrt(kT/m) rounded
                                          to a power of two, or a momentum sum of >= 64 particles within a factor two of
                                          the 32-bit range |sum v_d| < 512 u, or a cell with 2048 or more particles (the
                                          count and energy fields of the sweep's shared-memory sums hold fewer than 2048
                                          particles per cell; U19). 0 in every supported run              */
} mpc_obs;

/* Create a context. box[d] = L_d, cells[d] = number of fluid cells n_d; cells must be cubic
 * (L_x/n_x == L_y/n_y == L_z/n_z == a). n_per_cell = <N_c>, used for the virtual-wall-particle fill
 * (round(n_per_cell)) and for sizing. Allocates nothing on the device.
 * MPC_EINVAL: NULL argument, fewer than 3 cells along an axis, non-cubic cells, non-positive sizes/dt/kT/mass, rebin_every < 1,
 * brick dims not powers of two in 1..64 or tile too large for shared memory, more than one wall axis, force along a wall normal, walls with +a or MPC-AT
 * but without phantoms, phantoms without a no-slip wall, phantoms or solutes with rebin_every != 1 or with shear_rate, wall_velocity without a no-slip
 * wall on y or z,
 * SRD+a with thermostat (U6), MPC-AT with rebin_every != 1, key space >= 2^32, shear_rate != 0 with walls, MPC-AT or +a. */
int mpc_create(mpc_ctx** out, const float box[3], const int cells[3], float n_per_cell,
               const mpc_params* p, unsigned long long seed);

/* Number of keys K of the memory-order cell index (>= number of cells; brick padding and wall
 * layers included). Per-cell outputs of mpc_get_cells have K entries. */
int mpc_num_keys(const mpc_ctx*, unsigned long long* nkeys);

/* Current number of particles of the context: what mpc_set_state gave it; on a slab subdomain it changes when a reorder
 * hands particles over (after the step that completes the reorder). Size mpc_get_state's arrays with it. */
int mpc_num_particles(const mpc_ctx*, unsigned long long* n);

/* Bytes of device workspace needed for up to n_max particles. `compact` = 0: reorder through a
 * second copy of the particle arrays (fastest); 1: reorder property-wise through one 4-byte-per-
 * particle buffer, for systems where the second copy does not fit. */
int mpc_workspace_bytes(const mpc_ctx*, unsigned long long n_max, int compact, size_t* bytes);

/* Hand the library its workspace (device pointer, 256-byte aligned, `bytes` long, zeroing not
 * required) and the CUDA stream (a cudaStream_t cast to void*; NULL = legacy default stream).
 * The mode (compact or not) is chosen from `bytes`. MPC_ENOMEM if too small for n_max. The workspace must live
 * on the CUDA device that is current at the call (MPC_EINVAL otherwise); every later call on this context makes
 * that device current for its own duration. */
int mpc_bind(mpc_ctx*, void* workspace, size_t bytes, unsigned long long n_max, void* cuda_stream);

/* Copy a state in. Device pointers (mpc_set_state) or host pointers (mpc_set_state_host), n each.
 * id == NULL numbers the particles 0..n-1; ids given must be unique. `step` sets the step counter
 * t (the RNG streams depend on it). Positions must lie in [0, L_d) on periodic axes and in
 * [0, L_d] on the wall axis. Asynchronous on the bound stream. MPC_ESTATE on a slab subdomain between mpc_sub_begin
 * and mpc_sub_end or while a folded reorder is in flight (mpc_bind starts the context afresh). */
int mpc_set_state(mpc_ctx*, unsigned long long n, const float* x, const float* y, const float* z,
                  const float* vx, const float* vy, const float* vz, const unsigned* id, unsigned step);
int mpc_set_state_host(mpc_ctx*, unsigned long long n, const float* x, const float* y, const float* z,
                       const float* vx, const float* vy, const float* vz, const unsigned* id, unsigned step);

/* Advance nsteps MPC steps (nsteps >= 0). Asynchronous: only kernel launches and memsets on the
 * bound stream, no host synchronisation. Requires max |v| h < L/2 (single periodic wrap, U2).
 * One call of n steps gives bit-identical results to n calls of one step; it is faster because the
 * collision of step t is fused into the streaming pass of step t+1 and a reorder is folded into the
 * sweeps of its own and the next step.
 * The collision of the LAST step of a call stays pending inside the context: the next mpc_step applies it in its
 * first streaming pass, and every call that reads velocities (mpc_get_state*, mpc_observables) applies it first,
 * so the state seen through the API is always the fully collided one. */
int mpc_step(mpc_ctx*, int nsteps);

/* ---- slab subdomains (multi-GPU domain decomposition; one context per rank) ----------------------------
 * The step is split at its one exchange point. Every rank streams its own particles and adds their cell sums into
 * its own array; the sums of the cells in the four brick layers it shares with its two neighbours (its halo and first /
 * last own brick layer on either side) are ALSO added, inside the same kernel, into the neighbours' arrays with integer
 * reductions over peer memory (NVLink). Integer sums commute: after a barrier every rank holds the complete sums of
 * all its local cells, computes the same cell records from them as its neighbours do for the shared cells (the random
 * numbers are indexed by the cell's id in the whole box), and no particle is ever sent for a collision (the paper
 * exchanges the particles). The trajectory equals the single-GPU one bit for bit.
 * Particles change owner at the reorder, inside its kernels: the reorder of a subdomain is the one folded
 * into three sweeps; the particles whose cell of the reorder step lies in a halo layer are written by the
 * scatter pass straight into the new owner's staging buffer (peer memory), behind the owner's own particles of the cell;
 * the owner's read-back pass picks them up. This needs two further steps after the reorder step (steps_ahead below);
 * a reorder without them stays local (unfolded) and hands nothing over. mpc_sub_pack is the explicit alternative.
 *   mpc_sub_export   device pointers {cell sums, cell offsets, staging buffer (NULL: compact workspace)} and the local
 *                    brick-layer count of this rank, to hand to its neighbours
 *   mpc_sub_connect  the neighbours' pointers and layer counts (below = towards smaller z); clears the sums. The memory
 *                    must be reachable from this device (same device, or peer access / IPC mapping enabled by the caller).
 *                    A NULL staging pointer on either side (or a compact workspace here) turns the folded reorder off on this
 *                    rank; a rank that folds beside one that does not would write particles where nobody reads them, so if ANY
 *                    rank of the run exports no staging buffer the caller passes NULL for it on EVERY rank (slab_run.py does)
 *   mpc_sub_begin    MOVE + sums of the next step (+ the pending collision). steps_ahead = how many further
 *                    mpc_sub_begin calls the caller promises before it reads or replaces the state (mpc_get_state*,
 *                    mpc_observables, mpc_sub_pack, mpc_set_state*; MPC_ESTATE while a folded reorder is in flight);
 *                    all ranks must pass the same value. Then: barrier over all ranks. Whether a reorder is folded (and hands
 *                    particles over) is decided by every rank on its own, so it must come out the same everywhere: besides
 *                    steps_ahead, all ranks need the same mpc_set_debug flags, the same rebin_every, their mpc_set_state at the
 *                    same step, and staging buffers on all ranks or on none (mpc_sub_connect)
 *   mpc_sub_end      PROCESS_CELLS (+ the scan of a reorder). Then: barrier over all ranks. On the step of a folded reorder
 *                    this call synchronises the stream (it reads the rank's new particle count) and returns MPC_ENOMEM if the
 *                    hand-over would bring more particles than n_max: the context is then dead (every later call fails), and
 *                    the caller must keep EVERY rank from starting the next step, since that step's kernels of this rank and
 *                    of its neighbours write the arrivals into this rank's staging buffer (share the status at the barrier,
 *                    as slab_run.py does). All other mpc_sub_begin / mpc_sub_end calls only enqueue work
 *   mpc_sub_pack     between steps: the state split into the particles this rank keeps and those of its two neighbours
 * mpc_step returns MPC_ESTATE on a subdomain context. mpc_observables reports this rank's particles (kT_cell = 0). */
int mpc_sub_export(mpc_ctx*, void* device_ptrs[3], int* brick_layers);
int mpc_sub_connect(mpc_ctx*, void* const below[3], int brick_layers_below, void* const above[3], int brick_layers_above);
int mpc_sub_begin(mpc_ctx*, int steps_ahead);
/* Particles by owner ("sent to the new subdomain when the particles are sorted"), explicitly: applies the
 * pending collision, then copies the state into the seven DEVICE arrays (capacity: the current particle count each) class by
 * class: first the particles whose layer floor(z / a) is one of this rank's own, then those of the neighbour below,
 * then those of the neighbour above; counts[0..2] (host) = the three class sizes. Synchronises the stream. The caller
 * sends the two tails to the neighbours and gives mpc_set_state the particles it now owns. */
int mpc_sub_pack(mpc_ctx*, float* x, float* y, float* z, float* vx, float* vy, float* vz, unsigned* id,
                 unsigned long long counts[3]);
int mpc_sub_end(mpc_ctx*);

/* Diagnostic switches (change speed only, never results; the library reads no environment variables):
 * a bitwise OR of the flags below, 0 = the default code paths. May be called at any time between steps. */
#define MPC_DEBUG_NO_FUSE_GATHER  1u /* reorder: separate gather kernel instead of folding it into two sweeps      */
#define MPC_DEBUG_EAGER_CANONICAL 2u /* reorder: rank by id at every reorder instead of lazily on read             */
#define MPC_DEBUG_ATOMIC_SCATTER  4u /* reorder: cursor atomics per run of particles instead of the sweep's ranks   */
#define MPC_DEBUG_EAGER_COLLIDE   8u /* apply the last step's collision at the end of mpc_step (separate pass)      */
#define MPC_DEBUG_NO_LANE_SPREAD 16u /* reorder: plain cell order in memory instead of the lane-spread order (5a)  */
int mpc_set_debug(mpc_ctx*, unsigned flags);

/* Copy the state out, in the current internal order, with ids. Any pointer may be NULL (skipped).
 * Device pointers: asynchronous. Host pointers: synchronises the stream before returning.
 * Order: particles sorted by (memory key, id) as of the last reorder step (U3/U4).
 * The SRD hot path keeps the particles grouped by key only between reads (the order inside a cell does not
 * enter the physics: cell sums are integers); this call first restores the id order inside every cell
 * (a rank kernel and one gather on the bound stream), so what it returns is always the canonical order and
 * does not depend on how the steps were split over mpc_step calls. Calling it again costs only the copies. */
int mpc_get_state(mpc_ctx*, float* x, float* y, float* z, float* vx, float* vy, float* vz, unsigned* id);
int mpc_get_state_host(mpc_ctx*, float* x, float* y, float* z, float* vx, float* vy, float* vz, unsigned* id);

/* System observables ("Properties<FINALIZE>") into a HOST struct; synchronises.
 * profile_host: NULL, or n_profile host floats receiving the layer-averaged velocity component along the
 * force axis (first axis with g != 0, else x) as a function of the layer floor(r_w / a) along the
 * wall axis w (z if there is no wall), the shear-profile binning of PAPER.md:212. n_profile must equal the
 * number of fluid cells along that axis (MPC_EINVAL otherwise; ignored when profile_host is NULL).
 * Returns MPC_ERANGE (with *host_out filled in) if n_range_overflows != 0. */
int mpc_observables(mpc_ctx*, mpc_obs* host_out, float* profile_host, int n_profile);

/* ---- velocity profile for callers that cannot allocate device memory ------------------------------------------------
 * Everything above needs a workspace that the caller allocates and gives to mpc_bind. Some callers have no way to get
 * one: a monitoring or in-situ analysis hook that a host application calls from inside its time loop, where the
 * application's own caching allocator already owns almost all of the GPU's memory (a direct cudaMalloc fails there, and
 * where it does not, it stalls all streams of the device while it runs), code under a "nothing is allocated after
 * start-up" rule, or a caller that only holds pointers another runtime handed to it. This one call serves them. It needs
 * a context from mpc_create (host memory only; for the cell size a and the velocity unit of the fixed-point sums), no
 * mpc_bind and no workspace: its accumulation buffer is an array of fixed size inside the library image, 32 KiB of
 * device memory that every GPU which loads the library holds until the process exits.
 *
 * Computes, for the n particles given, the same quantity as mpc_observables' profile_host: for every
 * layer l = floor(r_w[i] / a) (clamped to 0 .. n_layers-1) the average of v_f[i] over the layer's particles, 0 for an
 * empty layer. The sums are 64-bit fixed point, so the result does not depend on the particle order and equals
 * mpc_observables' profile of the same particles bit for bit.
 *   r_w, v_f   DEVICE pointers, n floats each: the position component along the axis to bin over and the velocity
 *              component to average (e.g. z and vx as returned by mpc_get_state); may be NULL if n == 0. Not modified.
 *   profile    DEVICE pointer, n_layers floats, written by the call. counts: NULL, or a DEVICE pointer to n_layers
 *              64-bit unsigned integers receiving the number of particles per layer. The caller owns all four arrays.
 *   cuda_stream  a cudaStream_t cast to void* (NULL = legacy default stream); the call only enqueues work on it (one
 *              memset, two kernels) and does not synchronise: the outputs are valid once that work has completed.
 * All pointers must belong to the CUDA device that is current at the call, and the call runs there (it does not switch
 * to the device of mpc_bind). It calls no cudaMalloc, cudaFree or other allocating routine.
 * Limit: n_layers <= MPC_PROFILE_NOALLOC_MAX_LAYERS; more is refused with MPC_EINVAL (mpc_last_error says why) before
 * any CUDA call, and mpc_observables with a bound workspace is the way to go then. Also MPC_EINVAL: NULL context (no
 * message), n_layers < 1, NULL profile, NULL inputs with n > 0. MPC_ECUDA (sticky) if a CUDA call fails.
 * First call on a device: it looks up the device address of the built-in array (once per device and process, guarded by
 * a mutex). Make that first call before you start any stream capture.
 * Sharing: every call on a device, from any context, stream or thread, uses the same array, and the array keeps what the
 * last call left in it. Each call therefore clears the part it uses first, on its stream; two calls whose work overlaps
 * on the GPU (different streams without an ordering between them) race on the array and both results are garbage.
 * Calls on one stream, or ordered by events, are safe. */
#define MPC_PROFILE_NOALLOC_MAX_LAYERS 2048
int mpc_velocity_profile_noalloc(mpc_ctx*, unsigned long long n, const float* r_w, const float* v_f, int n_layers,
                                 float* profile, unsigned long long* counts, void* cuda_stream);

/* Test hook: the last step's pre-collision cell sums over real particles. Device pointers, any may
 * be NULL: count[K], px/py/pz[K] = m * sum v, e2[K] = sum |v|^2, key[n] = memory key of every
 * particle in the current order. Asynchronous. MPC_ESTATE before the first step. */
int mpc_get_cells(mpc_ctx*, unsigned* count, float* px, float* py, float* pz, float* e2, unsigned* key);

/* Test hook: one Philox-4x32-10 block computed by the library's generator (host side; the device
 * code uses the same function). */
void mpc_philox4x32_10(const unsigned ctr[4], const unsigned key[2], unsigned out[4]);

/* Number of kernel launches issued by this context so far (for bench.py's gpu_launches). */
unsigned long long mpc_launch_count(const mpc_ctx*);

/* Optional per-kernel-family timing with CUDA events recorded on the bound stream (bench.py's live
 * roofline measurement). mpc_profile_enable(ctx, 1) starts recording an event pair around every
 * kernel family of every following step (at most 16384 pairs between reads; later launches are
 * counted but not timed); mpc_profile_read synchronises the stream, returns for each of the
 * *n_families (<= 16) families its name, the summed device time in ms and the number of timed
 * sections since the last read, and resets the accumulators. Arrays are host pointers with room for
 * 16 entries; names point to static strings. */
int mpc_profile_enable(mpc_ctx*, int on);
int mpc_profile_read(mpc_ctx*, int* n_families, const char** names, double* total_ms, unsigned long long* launches);

const char* mpc_last_error(const mpc_ctx*);
int mpc_destroy(mpc_ctx*);

#ifdef __cplusplus
}
#endif
#endif /* MPC_B200_H */
