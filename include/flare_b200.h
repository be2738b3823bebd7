/*
 * flare_b200.h -- C ABI of libflare_b200.so: the per-timestep FLARE force-field evaluation
 * for molecular dynamics (arxiv 2204.12573), hand-written CUDA for sm_100a, FP64.
 *
 * Citations: "P:L<n>" = line n of the paper text; "R<k>" = reading k of
 * DESIGN.md section 3 (points where the paper is silent or garbled).
 *
 * What one evaluation computes, for every atom i:
 *   - its local environment rho_i: all neighbours within r_cut[s_i][s_j]          (R5,R6)
 *   - the ACE-B2 descriptor d_i: A[s,n,l,m] = sum_j T_n(2r/r_c-1) f_c(r) Y_lm(r^),
 *     B[nu1<=nu2,l] = sum_m A[nu1,l,m] A[nu2,l,m], d^_i = B/||B||                 (R1-R4)
 *   - the mapped mean  E_i = d^_i^T beta^(s_i)  d^_i                              (Eq. 1)
 *   - the mapped variance V_i = d^_i^T Sigma^(s_i) d^_i  (Sigma = the paper's gamma) (Eq. 2)
 *   - forces F = -grad sum_i E_i by the re-ordered summation that never forms
 *     grad d_i
 * and flare_step adds a velocity-Verlet NVE update (BASELINE.json north_star; R12).
 *
 * Conventions
 *   - Units: Angstrom, eV, amu, fs (R13).  a = KAPPA F/m with KAPPA = 9.648533212331e-3.
 *   - "device" pointers are CUDA device memory on the context's device; "host" pointers are
 *     ordinary host memory (pinned memory makes the *_host entry points faster, not different).
 *   - All arrays are dense, C-contiguous: positions/forces/velocities [N][3], matrices row-major.
 *   - The caller owns every array and the workspace; the library allocates device memory only
 *     in flare_create (model matrices and tables) and frees it in flare_destroy.
 *   - All device work is ordered on the stream given to flare_bind (inside an evaluation the launches of the small
 *     quadratic-form groups run on a library-owned side stream that forks from and joins back into it); device-pointer entry
 *     points are asynchronous (results valid after the caller synchronises that stream) unless
 *     stated otherwise.  *_host entry points and the flare_get_* hooks synchronise.
 *   - Results are in the CALLER's atom order although atoms are cell-sorted internally.
 *   - Every entry point returns FLARE_OK (0) or a negative FLARE_ERR_* code; nothing throws
 *     or aborts across this boundary.  flare_last_error() gives a message for the last failure.
 *   - There is no CPU fallback: without a CUDA device flare_create fails with FLARE_ERR_CUDA.
 */
#ifndef FLARE_B200_H
#define FLARE_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct flare_ctx flare_ctx; /* opaque, owned by the library */

enum {
    FLARE_OK = 0,
    FLARE_ERR_INVALID_ARG = -1,        /* null pointer, bad size, species out of range, asymmetric r_cut (R5) */
    FLARE_ERR_BOX_TOO_SMALL = -2,      /* a periodic box length < 2 max r_cut: no unique minimum image (R7) */
    FLARE_ERR_UNSUPPORTED_BOX = -3,    /* non-orthorhombic cell (R7) */
    FLARE_ERR_WORKSPACE_TOO_SMALL = -4, /* also: a domain-decomposition message, send list or capacity is too small */
    FLARE_ERR_NEIGHBOR_OVERFLOW = -5,  /* an atom has more than FLARE_OPT_MAX_NEIGHBORS neighbours */
    FLARE_ERR_CUDA = -6,               /* CUDA runtime error; message in flare_last_error */
    FLARE_ERR_NONFINITE = -7,          /* NaN/Inf met in positions, or produced in an energy, force or variance */
    FLARE_ERR_UNSUPPORTED = -8,        /* (n_max, l_max) outside the compiled range */
    FLARE_ERR_NOT_BOUND = -9,          /* call needs flare_bind / flare_set_state first */
    FLARE_ERR_HALO_EXCEEDED = -10      /* domain decomposition: an atom moved further since the last rebuild than the
                                          ghost shell covers (flare_domain_set_limit); forces since then are suspect */
};

/* Options (flare_set_option / flare_get_option).  Set them BEFORE flare_workspace_bytes/flare_bind. */
enum {
    FLARE_OPT_MAX_NEIGHBORS = 1, /* row stride of the neighbour table, 1..255 (default 48) */
    FLARE_OPT_CHUNK_ATOMS = 2,   /* atoms per chunk of the descriptor/quadratic-form/back-prop stage
                                    ("dividing atoms into batches"); 0 = automatic (default) */
    FLARE_OPT_TIMING = 3,        /* 1: bracket every kernel phase with CUDA events (flare_get_timings) */
    FLARE_OPT_SKIN_MILLI_ANGSTROM = 5, /* skin of the candidate neighbour list in 1e-3 Angstrom (default 400; 0 = off).
                                    With a skin the cell-sorted order and a list of all pairs within max r_cut + skin
                                    are kept across evaluations; every evaluation filters it with the exact predicate
                                    (R6, R12: the neighbour sets stay exact) and rebuilds it, on the device, as soon as
                                    two atoms of species a, b could have closed max r_cut + skin - r_cut[a][b] between
                                    them since the last build.  Candidate rows hold at most 64 entries
                                    (more: FLARE_ERR_NEIGHBOR_OVERFLOW; lower the skin).  Costs 360 B/atom. */
    FLARE_OPT_SKIN_REBUILDS = 6,  /* read-only (flare_get_option, synchronises): candidate-list rebuilds since flare_bind */
    FLARE_OPT_GRAPH = 7,          /* CUDA-graph replay of the MD step in flare_step / flare_step_nvt (small systems are bound by launch
                                    latency: one step of 256 atoms is ~30 tiny kernels).  -1 (default): automatic, for
                                    n_atoms <= 200 000 outside domain mode (there every ghost rebuild would force a
                                    re-capture); 0: never; 1: always.  The first step of a run (and the step after a
                                    re-bind, an option change or a new box) is launched plainly, the next one is captured
                                    -- with the candidate-list rebuild chain as a conditional IF node that a device-side
                                    decision switches on -- and later steps replay the graph on the bound stream.
                                    Results are bit-identical to plain launches.  Replayed steps record no phase timings. */
    FLARE_OPT_GRAPH_REPLAYS = 8,  /* read-only: steps replayed from the graph since flare_create */
    FLARE_OPT_SPECIES_SPARSE = 4 /* 1 (default when S * 2^S <= 64): atoms are grouped by the set of neighbour species
                                    present and the descriptor blocks of absent species are skipped in a2-a6
                                    ("420 to 112"); exact.  0: every atom uses all P components. */
};

/* Kernel phases reported by flare_get_timings, in this order. */
enum {
    FLARE_PHASE_NEIGHBOR = 0,   /* wrap, cell assign, sort, neighbour build, reverse-pair index  */
    FLARE_PHASE_DESCRIPTOR = 1, /* basis, A accumulation, B2 contraction, normalisation          */
    FLARE_PHASE_QFORM = 2,      /* beta and Sigma quadratic forms (FP64 DMMA grouped GEMM)        */
    FLARE_PHASE_BACKPROP = 3,   /* dE/dB -> dE/dA -> per-pair forces                              */
    FLARE_PHASE_GATHER = 4,     /* atomics-free force gather + E/V finalisation                   */
    FLARE_PHASE_INTEGRATE = 5,  /* velocity-Verlet kicks and drift                                */
    FLARE_N_PHASES = 6
};

/*
 * Create a model context (beta and gamma "computed ... once and stored").
 *   n_species  S >= 1
 *   mass_amu   [S] host, > 0
 *   n_max      radial functions per species (1..16); l_max angular cutoff (0..6)
 *   r_cut      [S*S] host, symmetric, > 0 (R5)
 *   beta       [S][P][P] host, row-major, eV; one matrix per CENTRAL species (R10); the
 *              library stores (beta + beta^T)/2, which leaves E unchanged.
 *   sigma      [S][P][P] host or NULL (then variances are unavailable); symmetrised likewise.
 *              P = N(N+1)/2 (l_max+1), N = S n_max (420 / 112 in the paper).
 *   cuda_device  ordinal; the context is tied to it.
 * The arrays are copied; the caller may free them after the call.  Synchronous.
 */
int flare_create(flare_ctx** out, int n_species, const double* mass_amu, int n_max, int l_max,
                 const double* r_cut, const double* beta, const double* sigma, int cuda_device);

void flare_destroy(flare_ctx* ctx);

/* Number of B2 descriptor components P for this context. */
int flare_num_descriptors(const flare_ctx* ctx);

int flare_set_option(flare_ctx* ctx, int option, int64_t value);
int flare_get_option(const flare_ctx* ctx, int option, int64_t* value);

/* Bytes of device workspace flare_bind needs for n_atoms atoms (0 on error). */
size_t flare_workspace_bytes(const flare_ctx* ctx, int64_t n_atoms);

/*
 * Attach a caller-owned device workspace (>= flare_workspace_bytes, 256-byte aligned) and the
 * CUDA stream (a cudaStream_t passed as void*; NULL = legacy default stream) all later work
 * runs on.  Re-binding with another n_atoms is allowed.  The workspace also holds the MD state.
 */
int flare_bind(flare_ctx* ctx, int64_t n_atoms, void* workspace, size_t bytes, void* cuda_stream);

/*
 * One force-field evaluation (steps a1-a8 of DESIGN.md).
 *   pos   [N][3] device, Angstrom, any image (wrapped internally, R6)
 *   types [N] device int32 in 0..S-1
 *   box   [9] host, row-major cell vectors; must be orthorhombic (R7)
 *   pbc   [3] host, non-zero = periodic
 *   e_out [N] device or NULL; f_out [N][3] device or NULL; var_out [N] device or NULL
 *         (NULL var_out skips the Sigma form entirely).
 * Asynchronous.  Device-detected failures (neighbour overflow, species out of range, non-finite input or
 * output) are reported by flare_check(), which synchronises; after such a failure the kept candidate list is
 * dropped, so the next evaluation starts from scratch.
 */
int flare_compute(flare_ctx* ctx, const double* pos, const int32_t* types, const double box[9],
                  const int pbc[3], double* e_out, double* f_out, double* var_out);

/* Same, HOST buffers: copies in, evaluates, copies out, synchronises, runs flare_check(). */
int flare_compute_host(flare_ctx* ctx, const double* pos, const int32_t* types, const double box[9],
                       const int pbc[3], double* e_out, double* f_out, double* var_out);

/* Synchronise the bound stream and return the first device-detected error of the work so far. */
int flare_check(flare_ctx* ctx);

/*
 * MD state (library-owned copy inside the workspace): positions, velocities [N][3] (Angstrom/fs),
 * types.  flare_set_state takes DEVICE pointers, flare_set_state_host HOST pointers.
 */
int flare_set_state(flare_ctx* ctx, const double* pos, const double* vel, const int32_t* types,
                    const double box[9], const int pbc[3]);
int flare_set_state_host(flare_ctx* ctx, const double* pos, const double* vel, const int32_t* types,
                         const double box[9], const int pbc[3]);

/*
 * Optional: supply the forces (eV/A, [N][3]) that belong to the state just set -- e.g. when resuming
 * from a checkpoint -- so that flare_step does not re-evaluate them before its first half-kick.
 * The caller vouches that they are the forces of those positions.  Device / host pointer versions.
 */
int flare_set_forces(flare_ctx* ctx, const double* f);
int flare_set_forces_host(flare_ctx* ctx, const double* f);

/*
 * n_steps of velocity Verlet (R12): v += dt/2 KAPPA F/m; x += dt v; wrap; F = F(x); v += dt/2 KAPPA F/m.
 * The neighbour list is rebuilt every step.  Forces of the current positions are evaluated
 * first if they are not yet valid.  want_variance != 0 also evaluates V_i each step.  Asynchronous.
 */
int flare_step(flare_ctx* ctx, double dt_fs, int n_steps, int want_variance);

/*
 * The same with a Nose-Hoover thermostat (the paper's production integrator; R19): every
 * step is bracketed by two thermostat half steps of length h = dt/2,
 *     xi += (h/2)(K2 - g kT)/Q ;  v *= exp(-xi h) ;  eta += xi h ;  xi += (h/2)(K2' - g kT)/Q,
 * K2 = sum m v^2 / KAPPA (eV), g = 3N - 3, Q = g k_B T tau^2, k_B = 8.617333262e-5 eV/K.  The thermostat state
 * (xi in 1/fs, eta) lives on the device (zeroed by flare_bind) and is read / set by the two calls below
 * (both synchronise).  Conserved: KE + sum E_i + Q xi^2/2 + g k_B T eta.  Asynchronous like flare_step.
 */
int flare_step_nvt(flare_ctx* ctx, double dt_fs, int n_steps, int want_variance, double T_kelvin, double tau_fs);
int flare_get_thermostat(flare_ctx* ctx, double* xi, double* eta);
int flare_set_thermostat(flare_ctx* ctx, double xi, double eta);

/*
 * Virial of the last evaluation (the model predicts "energy, forces and stress"):
 *     virial[3a+b] = dE/d eps_ab = sum_i sum_{j in N(i)} (dE_i/dr_ij)_a (r_ij)_b      (eV, symmetric),
 * reduced from the per-pair forces the evaluation stored; potential stress = virial / volume.  HOST output.
 * Synchronises.  Deterministic (fixed summation order).
 */
int flare_get_virial(flare_ctx* ctx, double virial[9]);

/*
 * The same virial for hosts that cannot allocate device memory and have no workspace to spare.
 *
 * Who needs it: a program that embeds this library and took all its device memory at start-up through its own pool
 * (at 10 M atoms that is nearly the whole 180 GB).  Inside such a program a cudaMalloc made on its behalf may find
 * nothing left, stalls every stream of the GPU while the driver maps memory (cudaFree does too), and is often simply
 * forbidden -- a pressure coupling or a monitor that runs every step has no room for either.  flare_get_virial
 * avoids allocation by taking its partial sums from the bound workspace and hands the result to the HOST after a
 * synchronisation; this call takes NOTHING from the caller but the result buffer, and leaves it on the device:
 *   virial_dev  [9] DEVICE doubles (row-major 3 x 3, eV), written by work enqueued on the bound stream;
 *               valid once the caller has synchronised that stream.  Asynchronous; no device error check
 *               (flare_check does that).
 * Its partial sums live in one array compiled into the library: FLARE_VIRIAL_STATIC_MAX_ATOMS / 2048 rows of 9
 * doubles = 147 456 bytes, held on every GPU that loads the library until the process ends, used or not.
 *   - Limit: a context bound to more than FLARE_VIRIAL_STATIC_MAX_ATOMS atoms is refused with FLARE_ERR_INVALID_ARG
 *     (flare_last_error names the limit); use flare_get_virial there.
 *   - The array is shared by every context and stream on a GPU.  Two calls that may run at the same time on one GPU
 *     (different streams, or contexts driven by different threads) corrupt each other's sums: order them yourself.
 *     Calls in sequence are safe -- each overwrites exactly the rows it then reads, so nothing left by the previous
 *     call is seen and nothing needs clearing.
 *   - The first call on each GPU looks up the array's device address (cudaGetSymbolAddress, with that GPU current;
 *     the runtime may load the library's kernels onto the GPU at that point).  Make that first call during set-up,
 *     before you begin any stream capture; later calls only launch two kernels.
 *   - It never calls cudaMalloc, cudaFree or any routine that allocates device memory, on any path.
 * Same preconditions as flare_get_virial (an evaluation has been run).  The sums are taken tile by tile (2048 atoms)
 * in a fixed order: repeated calls agree bit for bit; against flare_get_virial, whose order differs, to rounding.
 */
#define FLARE_VIRIAL_STATIC_MAX_ATOMS 4194304
int flare_virial_static(flare_ctx* ctx, double* virial_dev);

/*
 * On-the-fly analysis of the last evaluation, as in the paper's production run:
 *   max_unc     max_i sqrt(max(V_i, 0)) (the "maximum uncertainty"); n_above = #{i : sqrt(V_i) > unc_threshold}
 *               (both need an evaluation with variances, else FLARE_ERR_INVALID_ARG)
 *   coord       [N] device int32 or NULL: for atoms of species_a the number of neighbours of species_b with
 *               |r_ij| < r_coord (the paper: H atoms with another H within 1 A), 0 for other atoms;
 *               0 < r_coord <= r_cut[a][b] because the neighbour list is what is searched
 *   coord_hist  [16] host or NULL: histogram of those numbers over the species_a atoms (last bin: >= 15)
 * max_unc, n_above, coord_hist are HOST pointers; any output may be NULL.  Synchronises.
 */
int flare_analyze(flare_ctx* ctx, double unc_threshold, int species_a, int species_b, double r_coord,
                  double* max_unc, int64_t* n_above, int32_t* coord, int64_t* coord_hist);

/*
 * ---- Multi-GPU: spatial domain decomposition with a halo exchange per step (what the paper gets from LAMMPS:
 * P:L163 "MD runs entirely on GPUs with zero CPU-GPU data transfer except for I/O ... GPU-GPU communication";
 * near-perfect weak scaling P:L239; "near-two-dimensional" geometry P:L233).  One process per GPU owns the atoms
 * of one rectangle of a 2-D (x, y) process grid and evaluates them together with ghost copies of every atom within
 * the halo width h >= 2 max r_cut + 2 * (trigger displacement) of the rectangle, so that the forces on owned atoms
 * need no reverse exchange.  The library provides the DEVICE DATA PLANE: selection, packing, compaction and
 * unpacking kernels and every count live on the device; the caller only moves the message buffers between ranks
 * (e.g. NCCL send/recv) in the order below.  The state arrays of the context hold
 *     [ owned atoms ][ ghosts received in phase 0 (from lo, from hi) ][ ghosts received in phase 1 ]
 * in a LOCAL frame: a decomposed dimension is open (pbc = 0) with length w + 2 h and the owned rectangle at
 * [h, h + w); the frame of the neighbour on the lo side is shifted by +w, on the hi side by -w, so periodic images
 * need no special case.  Phase 0 exchanges along the first decomposed axis, phase 1 along the second and includes
 * the ghosts of phase 0 (corners).  Bind the context with the CAPACITY (owned + ghosts + slack) as n_atoms.
 *
 * Messages are device arrays of doubles: [0] = number of rows, rows start at double 8.  A full row is
 * (x, y, z, vx, vy, vz, fx, fy, fz, type, tag) = 11 doubles, a forward row (x, v, f) = 9 doubles; a message for
 * cap_rows rows needs 8 + 11 cap_rows doubles.  Messages of a REBUILD travel at full capacity with the count in the
 * header (no size round trip); forward messages have the sizes flare_domain_commit returned.
 *
 * Rebuild (every rank, same order):  [ per decomposed axis: migrate_pack -> exchange -> migrate_unpack ]
 *     [ per phase: border_pack -> exchange -> border_unpack ]  commit.
 * Step:  [ per phase: forward_pack -> exchange -> forward_unpack ]  flare_step(dt, 1, ...)  flare_domain_signal.
 * Between two rebuilds membership, order and counts are fixed, so the candidate neighbour list of the context is
 * kept (FLARE_OPT_SKIN_MILLI_ANGSTROM) and nothing blocks the host.  Ghosts carry their owner's velocity and force,
 * so flare_step moves them exactly as their owner does.  All calls are asynchronous on the bound stream except
 * flare_domain_begin and flare_domain_commit.  Too small a message, send list or capacity raises
 * FLARE_ERR_WORKSPACE_TOO_SMALL at the next flare_check / flare_domain_commit.
 */

/* Start domain mode: the first n_owned atoms of the state become pos / vel (may be NULL = 0) / types / tags (global
   atom ids, they travel with the atoms), all DEVICE pointers, in the local frame `box`, `pbc` (host).  A displacement
   of any atom by trigger_displacement (Angstrom) since the last rebuild raises the rebuild signal (0: always raised).
   If the call fails the context is left as it was.  While domain mode is active the whole-system calls
   (flare_compute*, flare_set_state*) are refused with FLARE_ERR_INVALID_ARG -- the context works on its local atoms,
   not on flare_bind's n_atoms; flare_bind ends domain mode. */
int flare_domain_begin(flare_ctx* ctx, int64_t n_owned, const double* pos, const double* vel, const int32_t* types,
                       const int64_t* tags, const double box[9], const int pbc[3], double trigger_displacement);

/* Owned atoms with coordinate[axis] < lo_bound (>= hi_bound) leave through the lo (hi) face: their full rows, shifted
   by shift_lo (shift_hi) along the axis, go to msg_lo (msg_hi); the atoms that stay are compacted in order.  Drops all
   ghosts. */
int flare_domain_migrate_pack(flare_ctx* ctx, int axis, double lo_bound, double hi_bound, double shift_lo,
                              double shift_hi, double* msg_lo, double* msg_hi, int64_t cap_rows);
/* Append the atoms of the two received messages (either may be NULL) to the owned set.  cap_rows is the capacity the
   messages were allocated for: a header count outside [0, cap_rows] (a peer built with another capacity, a stale
   buffer) is clamped to it and raises FLARE_ERR_WORKSPACE_TOO_SMALL at the next flare_check / flare_domain_commit;
   nothing is read beyond the message.  The same holds for flare_domain_border_unpack. */
int flare_domain_migrate_unpack(flare_ctx* ctx, const double* msg_lo_in, const double* msg_hi_in, int64_t cap_rows);

/* Phase 0 or 1: local atoms (owned, plus the ghosts of phase 0 in phase 1) with coordinate[axis] in [lo_a, lo_b)
   form the send list towards the lo neighbour, those in [hi_a, hi_b) the one towards the hi neighbour; their full
   rows (shifted) are packed.  The lists stay fixed until the next rebuild. */
int flare_domain_border_pack(flare_ctx* ctx, int phase, int axis, double lo_a, double lo_b, double hi_a, double hi_b,
                             double shift_lo, double shift_hi, double* msg_lo, double* msg_hi, int64_t cap_rows);
/* Append the ghosts received from the lo neighbour, then from the hi neighbour (NULL: none) and remember their slots. */
int flare_domain_border_unpack(flare_ctx* ctx, int phase, const double* msg_lo_in, const double* msg_hi_in,
                               int64_t cap_rows);

/* End of a rebuild (synchronises): the local atom count becomes the context's n_atoms, the candidate list is dropped,
   the rebuild signal cleared.  counts (host, may be NULL): [0] local atoms, [1] owned, [2..5] rows of the forward
   messages sent to x-lo, x-hi, y-lo, y-hi, [6..9] rows received from them, [10..13] their first slots. */
int flare_domain_commit(flare_ctx* ctx, int64_t counts[14]);

/* Per step: forward rows (x + shift, v, f) of the phase's two send lists -> messages; received rows -> ghost slots. */
int flare_domain_forward_pack(flare_ctx* ctx, int phase, double* msg_lo, double* msg_hi);
int flare_domain_forward_unpack(flare_ctx* ctx, int phase, const double* msg_lo_in, const double* msg_hi_in);

/* Copy the rebuild signal (0 / non-zero) of the last evaluation to a DEVICE int32: all-reduce it (MAX) over the ranks
   and rebuild when it is set.  Raised when an atom has moved trigger_displacement since the last rebuild. */
int flare_domain_signal(flare_ctx* ctx, int32_t* flag_out);

/* Copy the device-side error bits raised by the work enqueued so far (0 = none; what flare_check would turn into an
   error code) to a DEVICE int32, without synchronising and without clearing them.  A rank that hits an error would
   otherwise be the only one to know: reduce this (MAX) over the ranks together with the rebuild signal, and when the
   result is non-zero let EVERY rank call flare_check and stop, instead of leaving the peers blocked in an exchange. */
int flare_domain_status(flare_ctx* ctx, int32_t* status_out);

/* Guard of the ghost shell.  The rebuild that the signal asks for happens a few steps later (the flag is all-reduced
   and read with a lag), and until then the old shell is in use: it is complete only while no atom has moved more than
   half the halo skin since the last rebuild.  With max_displacement > 0 (Angstrom; it must exceed the trigger
   displacement) the kernel that tracks the displacements raises FLARE_ERR_HALO_EXCEEDED -- reported by the next
   flare_check / flare_domain_commit -- as soon as an atom has moved that far: owned atoms may have been missing
   dE_j/dr_jk terms since then, so the run should stop or restart from a checkpoint with a wider skin, a shorter lag or
   a smaller time step.  0 switches the guard off (the default after flare_domain_begin and flare_bind).  Like the
   signal it needs the candidate list (FLARE_OPT_SKIN_MILLI_ANGSTROM > 0).  Call after flare_domain_begin. */
int flare_domain_set_limit(flare_ctx* ctx, double max_displacement);

/* Global ids of the local atoms (owned first) -> DEVICE int64 [n_atoms]. */
int flare_domain_get_tags(flare_ctx* ctx, int64_t* tags_out);

/* Copy the state out; any pointer may be NULL.  Device-pointer version is asynchronous. */
int flare_get_state(flare_ctx* ctx, double* pos, double* vel, double* e, double* f, double* var);
int flare_get_state_host(flare_ctx* ctx, double* pos, double* vel, double* e, double* f, double* var);

/*
 * Test hooks (synchronise; HOST output pointers).
 * flare_get_neighbors: neighbour sets of the last evaluation in the caller's atom order, each
 *   row sorted by j; cnt [N], idx [N][stride] (entries past cnt[i] are -1).
 * flare_get_descriptors: re-evaluates the descriptors of the last evaluation's positions and
 *   returns B^ [N][P] and ||B|| [N] (caller's order).
 */
int flare_get_neighbors(flare_ctx* ctx, int32_t* cnt, int32_t* idx, int32_t stride);
int flare_get_descriptors(flare_ctx* ctx, double* bhat, double* nrm);

/*
 * Row statistics of the last evaluation's quadratic-form groups (synchronises; HOST outputs):
 * n_groups, and per group the number of atoms (rows) and of descriptor components it uses
 * (arrays of at least 64 entries).  The algorithmic flop count of steps a4/a5 is sum rows * 2 comps^2.
 */
int flare_get_groups(flare_ctx* ctx, int32_t* n_groups, int64_t* rows, int32_t* comps);

/*
 * Test hook (synchronises; HOST output): row[i] = quadratic-form row of atom i (caller's order) in the last
 * evaluation.  Rows are ordered by group; chunk c of step a8 holds rows [c * chunk, (c+1) * chunk) with
 * chunk = flare_get_option(FLARE_OPT_CHUNK_ATOMS), so tests can pick atoms next to a chunk boundary.
 */
int flare_get_rows(flare_ctx* ctx, int32_t* row);

/*
 * Accumulated CUDA-event time (ms) and launch count per phase since the last call
 * (needs FLARE_OPT_TIMING = 1); ms and launches are [FLARE_N_PHASES] host arrays.  Synchronises.
 */
int flare_get_timings(flare_ctx* ctx, double* ms, int64_t* launches);

/* Number of kernels the library has launched on this context since creation (steps replayed from a CUDA graph count
   the kernels of the captured step; those of its conditional rebuild chain, which run only on demand, are left out). */
int64_t flare_kernel_launches(const flare_ctx* ctx);

const char* flare_last_error(const flare_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* FLARE_B200_H */
