/*
 * hhrr.h -- C ABI of libhhrr: the fused HHRRLBM + wall-model time step on one B200.
 *
 * The calls follow the paper's statement of the problem (arxiv 2510.13726,
 * /root/reference/PAPER.md): a lattice of given extents, porosity and
 * solid velocity from a rotor description (Eq. 12-13 :133-140, Def. 1 :196-205,
 * Fig. 4 :254-269), wall-model cells at the porosity frontier (:157-188, :322-324),
 * the time loop of Listing 3 (:308-318), and as outputs the velocity moments (:147)
 * and the per-element integrated boundary force (Eq. 23 :211, :267, :315-317).
 *
 * Conventions.  D3Q27, dx = dt = 1, c_s^2 = 1/3.
 * Cell (x,y,z), linear index  x + nx*(y + ny*z)  (x fastest).  Direction
 * i = (cx+1) + 3(cy+1) + 9(cz+1), rest i = 13, opposite 26-i, weights
 * w_i = w(cx)w(cy)w(cz) with w(0)=2/3, w(+-1)=1/6.  Field arguments with several
 * components are SoA planes: u = [ux(all cells) | uy | uz].
 *
 * Memory.  Every pointer argument is a HOST pointer owned by the caller, unless its
 * name starts with d_ (device pointer, caller-owned).  The library allocates no
 * lattice-sized device memory: the caller hands hhrr_create() one device workspace
 * of at least hhrr_workspace_bytes() bytes (256-byte aligned), which the lattice
 * uses until hhrr_destroy(); the caller frees it afterwards.  All work is issued on
 * the CUDA stream given to hhrr_create (a cudaStream_t passed as void*; NULL = the
 * legacy default stream).  Calls that return data to host memory synchronise that
 * stream; hhrr_step() does not.
 *
 * Errors.  Every int-returning call returns HHRR_OK (0) or a negative hhrr_status
 * (hhrr_set_kernel_variant may also return the positive notice HHRR_W_FALLBACK);
 * nothing throws or aborts across the ABI.  hhrr_last_error() returns a
 * thread-local, NUL-terminated message for the last failing call on this thread.
 * There is no CPU fallback: without a usable CUDA device every call that needs one
 * fails with HHRR_E_CUDA.
 */
#ifndef HHRR_H_
#define HHRR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Velocity set of the library build: 27 = D3Q27 (default, libhhrr.so), 19 = D3Q19 (libhhrr_q19.so, the paper's
 * own lattice).  hhrr_velocity_set() tells which one a loaded library was built for.  D3Q19 holds
 * the directions of D3Q27 with |c|^2 <= 2 in the same order: rest i = 9, opposite 18 - i, weights 1/3, 1/18,
 * 1/36; every population buffer of the ABI then has 19 planes.                                              */
#ifndef HHRR_Q
#define HHRR_Q 27
#endif
#define HHRR_MAX_TAGS 16 /* element tags 1..15; tag 0 = none */

typedef enum {
  HHRR_OK = 0,
  HHRR_E_ARG = -1,   /* NULL / out-of-range argument                         */
  HHRR_E_SIZE = -2,  /* workspace too small or extents overflow int32 cells  */
  HHRR_E_CUDA = -3,  /* a CUDA runtime call or kernel launch failed          */
  HHRR_E_NAN = -4,   /* hhrr_check_finite found a non-finite population      */
  HHRR_E_STATE = -5, /* call not valid in the lattice's current state        */
  HHRR_W_FALLBACK = 1 /* not an error: hhrr_set_kernel_variant(5) on a lattice the default kernel cannot
                         tile -- the lattice keeps post-stream storage and variant 2 runs  */
} hhrr_status;

/* Outer boundary per axis (reading R12; the paper only names its outer
 * boundaries).  MIRROR = free-slip symmetry plane half a cell outside
 * the first / last cell: a population leaving through it returns to the same cell
 * with that velocity component reversed.                                            */
typedef enum { HHRR_PERIODIC = 0, HHRR_MIRROR = 1 } hhrr_axis_mode;

/* Cell types of Fig. 4 + the inflow fringe (R12). */
typedef enum {
  HHRR_FLUID = 0,    /* d = 1                                                     */
  HHRR_GROWTH = 1,   /* d = 1, one of the 26 neighbours has phi < eps/2 (:269)    */
  HHRR_FRONTIER = 2, /* |phi| < eps/2, 0 < d < 1  (Def. 1, Eq. 21-22 :196-203)    */
  HHRR_SOLID = 3,    /* phi <= -eps/2, d = 0                                      */
  HHRR_FRINGE = 4,   /* d = 0, u^B = u_in                                         */
  HHRR_BULK = 5      /* fluid outside the FSI region: bulk RRLBM-LES model (:215)  */
} hhrr_cell_type;

/* Half-open box of cells [x0,x1) x [y0,y1) x [z0,z1). */
typedef struct {
  int32_t x0, x1, y0, y1, z0, z1;
} hhrr_box;
#define HHRR_MAX_FSI_BOXES 8

typedef struct {
  int32_t nx, ny, nz;
  int32_t mode[3];           /* hhrr_axis_mode per axis                                       */
  double tau0;               /* molecular relaxation time, nu = c_s^2 (tau0 - 1/2)   (Eq. 14) */
  double sigma;              /* hybridisation factor of Eq. 7, in [0,1]        */
  double smagorinsky_cs;     /* C_S of Eq. 4                                 */
  double body_force[3];      /* g, lattice units (R11)                                        */
  double eps_cells;          /* transition width eps of Def. 1, in cells   */
  double kappa, E;           /* wall-function constants, 0.41 and 9.8          */
  int32_t newton_max_iter;   /* 10 in the paper                                */
  double newton_tol;         /* 1e-4 in the paper                              */
  double sampling_distance;  /* h_s: wall-model sampling distance along the normal, in cells  */
} hhrr_params;

/* "Rotor description": a rotor-frame reference grid of signed distances (the paper
 * keeps it at twice the lattice resolution) with an element tag
 * per node (:267), rotating rigidly (:265) about `axis` (unit vector) through
 * `centre` at `omega` rad per step from angle `theta0`.  Node (ix,iy,iz) sits at
 * rotor-frame position origin + spacing*(ix,iy,iz) relative to the centre, and at
 * index ix + gx*(iy + gy*iz).  sdf/tag are read during hhrr_set_rotor only.      */
typedef struct {
  const float* sdf;
  const uint8_t* tag;
  int32_t gx, gy, gz;
  double spacing;
  double origin[3];
  double centre[3], axis[3], omega, theta0;
  int32_t n_tags; /* tags 1..n_tags are rotor elements (blades, hub) */
} hhrr_rotor_desc;

typedef struct hhrr_lattice hhrr_lattice; /* opaque, owned by the library */

/* Device bytes hhrr_create needs for `p` (and, if rotor != NULL, for that rotor's
 * reference grid).  Returns 0 on invalid arguments.                                 */
size_t hhrr_workspace_bytes(const hhrr_params* p, const hhrr_rotor_desc* rotor);

/* Creates a lattice at rest (f_i = w_i, d = 1, no geometry) in the caller's device
 * workspace.  `cuda_stream` is a cudaStream_t: every kernel and copy of the library is
 * queued on it, except two things hhrr_step puts on one internal side stream, ordered against
 * `cuda_stream` by events: the porosity update of the NEXT step (a function of the step count
 * only; written into an alternate geometry set) and the force collection of the
 * step just streamed (it only reads).  hhrr_step returns with the side stream joined into
 * `cuda_stream`.  Results do not depend on it (hhrr_set_lookahead(L, 0) switches the look-ahead
 * off, for measurement and tests).  The workspace must stay allocated until hhrr_destroy,
 * which waits for both streams.                                                           */
int hhrr_create(const hhrr_params* p, void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                hhrr_lattice** out);
int hhrr_destroy(hhrr_lattice* L);

/* f = f_eq(rho,u) (Eq. 11); with_neq != 0 adds the regularised
 * f^(1) of Eq. 8-10 with a1^(2) = -2 rho c_s^2 tau0 S^FD(u).  rho: N, u: 3N floats. */
int hhrr_init_equilibrium(hhrr_lattice* L, const float* rho, const float* u, int with_neq);

/* Static geometry as a signed-distance field phi (N floats; > 0 fluid).  Types and
 * porosity follow Def. 1 from phi; tag (N bytes, nullable = all 1) names the element;
 * d_override (N floats, nullable) replaces the linear ramp of Eq. 22 inside the
 * transition band (e.g. a tanh ramp).  phi == NULL removes the static geometry.     */
int hhrr_set_static_geometry(hhrr_lattice* L, const float* phi, const uint8_t* tag,
                             const float* d_override);
/* Rigid-body velocity of element `tag`: u^B(x) = vel + omega x (x - centre). */
int hhrr_set_body(hhrr_lattice* L, int32_t tag, const double centre[3], const double omega[3],
                  const double vel[3]);
/* Inflow fringe (R12): cells with x_begin <= x < x_end get d = 0, u^B = u_in. */
int hhrr_set_fringe(hhrr_lattice* L, int32_t x_begin, int32_t x_end, const double u_in[3]);
/* Region split of PAPER.md:215 ("a simpler RRLBM-LES model is applied for all parts of the domain
 * that are guaranteed to not intersect the moving wall-modeled structures", Listing 2 :271-302;
 * DESIGN.md R20).  `boxes` (host, n_boxes <= HHRR_MAX_FSI_BOXES, copied) name the FSI part of the
 * lattice; a FLUID cell outside every box becomes HHRR_BULK and collides with the bulk model: plain
 * momentum, third-order recursive-regularised collision with the Smagorinsky relaxation, no hybrid
 * finite-difference part (Eq. 7 at sigma = 1).  Blocks of the collide-stream kernel that hold only
 * bulk cells then need no neighbour velocities at all.  Every cell that is not plain fluid (solid,
 * frontier, growth, fringe) must lie inside a box: if one does not, its type is kept and
 * hhrr_check_finite returns HHRR_E_STATE.  n_boxes = 0 (default): HHRRLBM everywhere.          */
int hhrr_set_fsi_region(hhrr_lattice* L, int32_t n_boxes, const hhrr_box* boxes);
/* Wall function solved by the wall model: 0 = the paper's truncated Spalding law (Eq. 18, PAPER.md:172;
 * default), 1 = Musker's explicit profile u+ = 5.424 atan((2y+ - 8.15)/16.7) + log10((y+ + 10.6)^9.6 /
 * (y+^2 - 8.15 y+ + 86)^2) - 3.52 (BASELINE.json config 3 "Spalding/Musker"), solved as
 * U/u_tau = u+(y u_tau/nu) with the same Newton iteration and stop rule (Eq. 19).  */
int hhrr_set_wall_function(hhrr_lattice* L, int32_t kind);
/* Second readings of the two wall-model passages the paper leaves open.
 * slip  0 (default): the friction velocity is added to the porous-medium velocity, u_wm = u_tau e_t
 *                    ("adding it to the velocity moment of the porous medium");
 *       1          : the wall-function velocity at the cell's own wall distance y1 ("wall modelled
 *                    velocities ... at Y1", :314): u_wm = u_tau u+(y1 u_tau/nu) e_t, u+ the selected wall
 *                    function (the inverse of Eq. 17, :166, by Newton; Musker's profile is explicit).
 * shear 0 (default): one-sided difference between the sampling point and the cell,
 *                    G = (v_s - v(x_w)) n^T / h_s (:324);
 *       1          : analytic slope of the wall function at the sampling point ("shear stress (cf. Eq. 17)"),
 *                    G = du/dy e_t n^T, du/dy = (u_tau^2/nu) du+/dy+.            S_wm = (G + G^T)/2 in both.
 * Takes effect from the next step.  HHRR_E_ARG for other values.                                          */
int hhrr_set_wall_model_variant(hhrr_lattice* L, int32_t slip, int32_t shear);
/* Rotor (copied to the device workspace); sets the bodies of tags 1..n_tags. */
int hhrr_set_rotor(hhrr_lattice* L, const hhrr_rotor_desc* rotor);
/* Wall model on the cells {FRONTIER, phi > 0} (R13). */
int hhrr_enable_wall_model(hhrr_lattice* L, int enable);
/* Evaluates geometry(current step) now (InitializePorosityO). */
int hhrr_update_geometry(hhrr_lattice* L);

/* n_steps passes of Listing 3: UpdatePorosityO, collide & stream
 * (Eq. 6-14), WallModelO, boundary-force collection and per-element integration,
 * rigid rotation.  Asynchronous on the lattice's stream.                            */
int hhrr_step(hhrr_lattice* L, int32_t n_steps);
int64_t hhrr_step_count(const hhrr_lattice* L);

/* rho (N) and v = (j + g/2)/rho (3N, SoA) of the current populations. */
int hhrr_get_moments(hhrr_lattice* L, float* rho, float* v);
/* Same, into DEVICE buffers, asynchronous on the stream (no host copy). */
int hhrr_get_moments_device(hhrr_lattice* L, float* d_rho, float* d_v);
/* Force ON each element per step, F[(s - first_step)*HHRR_MAX_TAGS*3 + tag*3 + a],
 * for steps first_step .. first_step+n_steps-1 (must lie within the last
 * hhrr_force_history() steps taken).                                                */
int hhrr_get_forces(hhrr_lattice* L, int64_t first_step, int64_t n_steps, double* F);
/* Torque ON each element per step about the centre of the element's rigid body (hhrr_set_body):
 * M_k = sum over the cells x of element k with d < 1 of (x - x_c) x F(x), F(x) the cell's
 * momentum-exchange force of Eq. 23 as summed by hhrr_get_forces.  The paper
 * integrates forces only; the torque is SURVEY 8(f)-4's output for torque / power coefficients.
 * Same layout, history and error behaviour as hhrr_get_forces; M is a HOST buffer.            */
int hhrr_get_torques(hhrr_lattice* L, int64_t first_step, int64_t n_steps, double* M);
/* Thrust coefficient, Definition 3 / Eq. 26: C_T = T / (0.5 rho pi r^2 U_inf^2), T = "the integral
 * of all axial forces acting on the rotor" = sum over the rotor's elements (tags 1..n_tags of hhrr_set_rotor) of
 * F_k . a, with F_k of hhrr_get_forces and a the unit rotor axis -- and, from the torques of the same elements, the
 * power coefficient C_P = (sum_k M_k . a) omega / (0.5 rho pi r^2 U_inf^3) (the paper reports C_T
 * only).  rho, u_inf, radius: lattice units, all > 0 (HHRR_E_ARG otherwise).  c_t, c_p: HOST arrays of n_steps
 * doubles, one value per step, either may be NULL.  Steps as for hhrr_get_forces; HHRR_E_STATE without a rotor.
 * Host arithmetic on the recorded forces: synchronises the stream.                                                  */
int hhrr_get_rotor_coefficients(hhrr_lattice* L, int64_t first_step, int64_t n_steps, double rho, double u_inf,
                                double radius, double* c_t, double* c_p);
int64_t hhrr_force_history(void);
/* Cell types / tags / porosity of the last evaluated geometry (any pointer nullable). */
int hhrr_get_cell_types(hhrr_lattice* L, uint8_t* type, uint8_t* tag, float* d);
/* Wall-model cell list in ascending cell index.  *count receives the list length;
 * at most `capacity` entries are written.  idx: cell index; y1n: 3 doubles per entry
 * (wall distance times unit normal); u_tau: last friction velocity;
 * valid: 1 if the cell carries a wall-model state -- only then is u_tau ever read (the
 * Newton warm start; a cell without state starts from Eq. 20); what the array keeps for a
 * cell without state is history.  Array pointers nullable.                            */
int hhrr_get_wall_list(hhrr_lattice* L, int64_t capacity, int32_t* idx, double* y1n, double* u_tau,
                       uint8_t* valid, int64_t* count);
/* Wall-model output of one cell: slip velocity u_wm[3] and strain S_wm[6] (xx yy zz xy xz yz). */
int hhrr_get_wall_state(hhrr_lattice* L, int64_t cell, double* u_tau, double u_wm[3], double s_wm[6],
                        int32_t* valid);
/* Populations as stored: deviations f_i - w_i, 27 planes of N floats.
 * Checkpoint / resume: the state of a run is (step count, populations, wall-model state); the geometry is a
 * function of the setters' inputs and the step count.  To resume: create the lattice, call the same setters,
 * then hhrr_set_step_count, hhrr_set_populations, hhrr_set_wall_model_state (in this order).  The run then
 * continues bitwise as the uninterrupted one (forces of earlier steps are not part of the state).        */
int hhrr_get_populations(hhrr_lattice* L, float* f_minus_w);
int hhrr_set_populations(hhrr_lattice* L, const float* f_minus_w);
/* Wall-model state of the cells of the current wall list, in list order: cell index, u_tau (the Newton warm
 * start, Eq. 20), slip velocity u_wm[3 per cell], strain S_wm[6 per cell: xx yy zz xy xz yz] as
 * stored (fp32), valid flag.  *count = number of wall cells; nothing else is written if capacity < *count.   */
int hhrr_get_wall_model_state(hhrr_lattice* L, int64_t capacity, int32_t* idx, double* u_tau, float* u_wm, float* s_wm,
                              uint8_t* valid, int64_t* count);
/* Restores it: evaluates the geometry of the current step if needed (as hhrr_update_geometry does: state of cells
 * outside its wall-model set is dropped), then writes the state of every listed cell that belongs to that set
 * (others are ignored).  Save a checkpoint from an evaluated state -- after a step, or after hhrr_update_geometry
 * when a setter was called since -- and restore it under the same setters: the run then continues as above.      */
int hhrr_set_wall_model_state(hhrr_lattice* L, int64_t count, const int32_t* idx, const double* u_tau, const float* u_wm,
                              const float* s_wm, const uint8_t* valid);
/* Sets the step counter (rotor angle theta0 + step * omega; slot of the force ring). */
int hhrr_set_step_count(hhrr_lattice* L, int64_t step);
/* Populations (deviations f_i - w_i) of selected cells: out[k*27 + i] for cells[k], and the
 * cells' flags as stored (type | tag << 3 | wall-model-valid << 7) if flags != NULL.  Lets tests
 * check sampled cells of lattices too large to copy back whole.                          */
int hhrr_get_cell_populations(hhrr_lattice* L, int64_t n_cells, const int64_t* cells, float* out,
                              uint8_t* flags);
/* Time-n homogenised velocity field of the last collide (3N floats), for tests.  Only the two-pass kernel
 * (variant 0) stores it; HHRR_E_STATE otherwise or before the first step.                    */
int hhrr_get_uhat(hhrr_lattice* L, float* uhat);
/* Slab decomposition along z (the paper's multi-GPU layout: one block per GPU).  A rank's
 * lattice is z-periodic and holds one HALO plane at either end (z = 0, z = nz - 1) around its nz - 2 real planes.
 * After every hhrr_step(L, 1) the ranks exchange, per face, hhrr_halo_floats(L) floats:
 *   hhrr_halo_pack(L, face, d_buf)    face 0 = low z, 1 = high z; asynchronous on the stream: the populations the
 *                                     collision pushed into the halo plane (they belong to the neighbour's first real
 *                                     plane) and the other populations of the last real plane (the neighbour's halo);
 *   hhrr_halo_unpack(L, face, d_buf)  at the RECEIVING rank with the face the data arrived through, i.e. the buffer
 *                                     a neighbour packed with face 1 is unpacked with face 0 and vice versa.
 * d_buf is a device pointer (it may be peer-mapped memory of the neighbour GPU: the pack kernel's stores then are
 * the transfer).  Structures (cells with d < 1 and their wall-model stencils) must stay clear of the halo planes
 * and the planes next to them; the fringe and plain fluid may cross.  The exchanged state equals the undecomposed
 * lattice's bit for bit (tests/test_slabs*.py).                                                                  */
int64_t hhrr_halo_floats(const hhrr_lattice* L);
int hhrr_halo_pack(hhrr_lattice* L, int32_t face, float* d_buf);
int hhrr_halo_unpack(hhrr_lattice* L, int32_t face, const float* d_buf);
/* Allocation-free wall model, for callers that may not allocate (CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc).  Runs WallModelO (Listing 3 line 4; Eq. 15-20 :159-184) on the lattice's CURRENT
 * populations and the wall list of the last evaluated geometry -- what the wall model inside the last hhrr_step saw --
 * asynchronously on the lattice's stream, and writes its results per LIST ENTRY e (order of hhrr_get_wall_model_state)
 * into caller-owned DEVICE arrays instead of the lattice's state, which it neither reads nor writes:
 *   d_u_tau_start  [capacity] doubles or NULL: warm start of the Newton iteration per entry (Eq. 20 :181); <= 0 or NULL =
 *                  the cold start sqrt(nu U / y);
 *   d_u_tau [capacity] doubles, d_u_wm [capacity][3] floats, d_s_wm [capacity][6] floats (xx yy zz xy xz yz).
 * Entries [0, min(wall count, capacity)) are written.  The scratch between its two kernels (48 B per wall cell) is a
 * file-scope device array of HHRR_NOALLOC_MAX_WALL_CELLS cells = 3 MiB that every GPU which loads the library holds
 * until exit: capacity > HHRR_NOALLOC_MAX_WALL_CELLS is refused with HHRR_E_SIZE.  The call allocates and frees nothing
 * and does not synchronise.  All calls share the scratch: calls that overlap on one GPU (different streams) race; calls
 * on one stream or on different GPUs do not.  Nothing in the scratch needs clearing between calls.                    */
#define HHRR_NOALLOC_MAX_WALL_CELLS 65536
int hhrr_wall_model_noalloc(hhrr_lattice* L, int64_t capacity, const double* d_u_tau_start, double* d_u_tau,
                            float* d_u_wm, float* d_s_wm);
/* HHRR_E_NAN if any population is non-finite (synchronises). */
int hhrr_check_finite(hhrr_lattice* L);
/* Selects the collide-stream kernel: 5 = the TMA-fed fused kernel on x-pull / yz-push storage
 * (default; needs a periodic x axis and tiles of 64 x 8 cells (nx % 64 == 0, nx >= 128,
 * ny % 8 == 0) or 128 x 4 cells (nx % 128 == 0, nx >= 256, ny % 4 == 0)); 2 = the fused
 * warp-specialised kernel on post-stream storage (any extents, any axis modes); 0 = two-pass
 * (moments pass + collide pass; the bring-up path the fused kernels were checked against).
 * All compute the same step (Listing 3 line 3).  Variant 5 keeps plane i of
 * the population buffer as f_i(x + c_ix, y, z) (the x move of Eq. 6, is taken on
 * the read side); the call re-stores the current populations when the layout changes, and
 * every entry point that takes or returns populations speaks the plain post-stream layout.
 * Returns HHRR_W_FALLBACK (> 0, hhrr_last_error() says why) when 5 is asked for on a lattice
 * it cannot tile: variant 2 then runs; hhrr_create makes the same choice silently, and
 * hhrr_population_storage tells which kernel a lattice runs.                              */
int hhrr_set_kernel_variant(hhrr_lattice* L, int32_t variant);
/* 1 if the populations are currently kept x-pulled (variant 5 running its own kernel), 0 if
 * post-stream (all other variants, and variant 5 on a lattice it cannot tile).            */
int hhrr_population_storage(const hhrr_lattice* L);
/* Optional CUDA-event timing of the collide-stream launches inside hhrr_step (the kernel the
 * roofline is quoted on).  hhrr_get_timing synchronises, returns the summed device time in
 * milliseconds and the number of launches it covers (at most 1024 per window), and starts a
 * new window.  (The first hhrr_set_timing(L, 1) creates 2048 CUDA events, the only device-side resources besides
 * a side stream and a handful of ordering events that the library creates itself; hhrr_destroy releases them.)          */
int hhrr_set_timing(hhrr_lattice* L, int enable);
/* Launch shape of the default kernel (variant 5): planes per z-chunk of a tile column and tiles per thread-block
 * cluster (1, 2, 4, 8).  0 = automatic (16 planes, 12 with an FSI region; 40 / 22 on D3Q19; clusters of 2: measured on config 5,
 * profiles/r02_k2_chunk_scan.md).  Results do not depend on it; it exists so that the scan behind the defaults can be
 * repeated (bench.py --chunk-planes / --cluster).                                                               */
int hhrr_set_launch_shape(hhrr_lattice* L, int32_t chunk_planes, int32_t cluster);
/* Switches the overlap of the next step's porosity update with the current step (see
 * hhrr_create) on (default) or off.  Results are bitwise the same either way.            */
int hhrr_set_lookahead(hhrr_lattice* L, int enable);
int hhrr_get_timing(hhrr_lattice* L, double* ms_collide_stream, int64_t* launches);
/* Number of kernel launches issued by this lattice so far. */
int64_t hhrr_launch_count(const hhrr_lattice* L);

const char* hhrr_last_error(void);
const char* hhrr_version(void);
int32_t hhrr_velocity_set(void);

#ifdef __cplusplus
}
#endif
#endif /* HHRR_H_ */
