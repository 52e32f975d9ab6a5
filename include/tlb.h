/*
 * tlb.h -- C ABI of the B200-native thermal two-component D2Q9 lattice-Boltzmann step.
 *
 * The operation is the per-time-step update of TLBfind (arXiv 2109.12565); citations are
 * "PAPER L<line>" into /root/reference/PAPER.md plus the equation / section they fall in.
 * Readings R1..R32 of silent or garbled passages are listed in DESIGN.md.
 *
 * One step (tlb_step) computes, for every fluid site, from time-t populations only (R13):
 *   moments            rho_l = sum_i f_l,i ; T = sum_i g_i ; j = sum_l,i c_i f_l,i     Eqs. (4),(5),(17) L76-80, L165
 *   pseudopotentials   psi^x = rho/rho0 ; psi^s = rho0 (1 - exp(-rho/rho0))            Eqs. (8),(12) L114, L131
 *   forces             cross (NN, w_i), attractive (NN, w_i), repulsive (NN+NNN, p_i)   Eqs. (7),(10),(11) L89, L123-126
 *   buoyancy           F_l,y += rho_l alpha_g (T - T_ref)                               Eq. (22), footnote L182
 *   velocities         u = j/rho ; u_l = u + tau F_l/rho_l ; u^(H) = (j + F/2)/rho      Eqs. (5),(6) L78-84; L139
 *   BGK collision      f_l (rho_l, u_l, tau) ; g (T, u^(H), tau_g)                      Eqs. (2),(3),(16),(18) L67-71, L161-169
 *   streaming          f_i(x + c_i, t+1) = f*_i(x, t), x periodic                      Eq. (1)
 *   walls / obstacles  half-way bounce-back for f (L151), anti-bounce-back at the wall
 *                      temperature for g (L314, R8), wall densities in the force
 *                      stencil (L155, R9); done by a separate boundary kernel.
 *
 * CONVENTIONS
 *   Lattice: nx x ny sites, x periodic (L147); y bounded by walls whose half-way planes are at
 *   y = -1/2 and y = ny - 1/2 (API rows y = 0..ny-1 are the paper's fluid rows 1..ny, L155), or
 *   periodic if params.periodic_y.
 *   Layout: every field is row-major [ny][nx], x fastest; `u` is [2][ny][nx] (u^(H)_x plane then
 *   u^(H)_y); a population set is [9][ny][nx] in the direction order (R1)
 *     i : 0      1      2      3       4       5      6       7        8
 *     c : (0,0)  (1,0)  (0,1)  (-1,0)  (0,-1)  (1,1)  (-1,1)  (-1,-1)  (1,-1)
 *   and holds the time-t (post-streaming, pre-collision) populations f_i(x, t); solid sites hold 0.
 *   Solid sites report rho = rho_wall, u = 0, T = T_bottom in the lower half and T_top in the upper.
 *   Pointers: every array argument of the un-suffixed calls is a DEVICE pointer owned by the caller;
 *   the *_host variants take HOST pointers (pinned memory makes the copies asynchronous) and stage
 *   through the workspace.  Nothing is retained from any argument after the call returns, except
 *   `workspace` and `stream` given to tlb_create, which must outlive the handle.
 *   Asynchrony: device-pointer calls enqueue on the handle's stream and return; *_host calls and
 *   tlb_observables_host return after the stream has been synchronised.
 *   Errors: every call returns 0 (TLB_OK) or a negative code, never aborts or throws.  A CUDA error raised by
 *   the handle's own work is sticky on the handle (TLB_ECUDA from then on).  A CUDA error that some other
 *   library left pending on the calling thread makes a call return TLB_ECUDA without doing anything and
 *   without consuming or adopting that error.
 *   Device: the handle lives on the CUDA device that owns `workspace`; every entry point makes that device
 *   current for its duration and restores the caller's, so a multi-GPU host process may switch devices freely.
 *   `stream` must be a stream of that device.
 *   There is no CPU fallback: without a CUDA device tlb_create returns TLB_ECUDA.
 *
 * Y-SLABS (multi-GPU, the paper's stated future work L376)
 *   tlb_create_slab makes a handle for rows [y0, y1) of an nx x ny lattice.  Its local lattice has
 *   ny_local = (y1 - y0) + halo_lo + halo_hi rows: 3 halo rows beyond every face that is not a flat wall of
 *   the whole lattice (with periodic_y every face has them and row indices wrap).  Every array argument of a
 *   slab handle is [ny_local][nx] (or [9][ny_local][nx]), local row r being row (y0 - halo_lo + r) of the
 *   whole lattice; state-setting calls take the halo rows from the caller's arrays, output calls write the
 *   owned rows only.  One time step is
 *       tlb_slab_step_edges     fused kernel on the 3 owned rows next to each halo face
 *       tlb_slab_step_interior  fused kernel on the remaining owned rows (overlaps the exchange)
 *       ... the caller moves the 3 edge rows of each face into the neighbour's halo rows ...
 *       tlb_slab_step_finish    boundary kernel over every solid node of the local lattice; state advances
 *   The default transport is zero-copy: the 27 plane rows of a lattice row lie next to one another, so the rows to
 *   export and the halo rows to fill are each ONE contiguous block of tlb_halo_bytes inside the population buffer, and
 *   tlb_halo_region(face, which) returns their device pointers for NCCL send / recv, a peer copy or a peer-mapped
 *   store to read and write directly.  tlb_halo_pack(face) / tlb_halo_unpack(face) copy the same rows to / from a
 *   separate buffer for transports that want one (the staged alternative; both give bit-identical states).
 *   (3 rows: the pull of the 2 force-stencil rows beyond a face reaches one row further.)  The result is bit
 *   for bit that of one handle on the whole lattice.  tlb_observable_sums gives a slab's share of the six
 *   sums behind tlb_observables; after an all-reduce tlb_observables_from_sums finishes them.
 */
#ifndef TLB_H
#define TLB_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  TLB_OK = 0,
  TLB_EINVAL = -1,     /* bad size / parameter / NULL pointer / workspace too small              */
  TLB_ESTATE = -2,     /* step / fields / observables before any state was set                   */
  TLB_ECUDA = -3,      /* a CUDA call failed (sticky on the handle); see tlb_last_cuda_error      */
  TLB_EPLACEMENT = -4, /* tlb_init could not place n_droplets within 1000 * n_droplets candidates */
  TLB_EIO = -5,        /* a checkpoint file could not be opened, or has the wrong size              */
  TLB_ELIMIT = -6      /* a size beyond the fixed capacity of tlb_t1_events_static                 */
};

/* POD, passed by pointer, copied by tlb_create. */
typedef struct tlb_params {
  double tau, tau_g;                  /* relaxation times, Eqs. (2),(16); must be > 0.5 (Eqs. (14),(20))   */
  double rho0;                        /* reference density of Eqs. (8),(12); > 0                            */
  double G12, G11a, G11r, G22a, G22r; /* couplings of Eqs. (7),(10),(11); G*a < 0 attractive, G*r > 0      */
  double rho_wall_A, rho_wall_B;      /* densities seen by the force stencil at solid nodes, L155 (R9)      */
  double T_bottom, T_top, T_ref;      /* wall temperatures L314; buoyancy reference, footnote L182 (R12)    */
  double alpha_g;                     /* alpha*g of Eq. (22)                                                */
  double body_ax;                     /* EXTENSION: uniform acceleration along x (Poiseuille test)          */
  double u_wall_bottom, u_wall_top;   /* x-velocity of the flat walls (Couette, L147-151, Eq. (15); R20)    */
  /* input recipe used by tlb_init only */
  double droplet_radius, min_gap, rho_in, rho_out, noise_amp;
  int32_t n_droplets;
  int32_t periodic_y;                 /* 0: walls (default); 1: periodic in y (L147, L284-302)              */
  int32_t thermal;                    /* THERMAL switch, L314: 0 leaves g untouched (the step neither reads */
                                      /* nor writes it) and the buoyancy uses T = T_ref; tlb_fields and Nu  */
                                      /* still report sum_i g_i of the frozen populations                   */
  int32_t post_w, post_h, post_period;/* structured rough walls used by tlb_init (R19); 0,0,0 = smooth      */
  int32_t pop_precision;              /* storage of the populations in HBM: 64 (default) or 32 (bandwidth   */
                                      /* study of BASELINE config 5; the arithmetic stays fp64)             */
  int32_t reserved;
} tlb_params;

typedef struct tlb_handle tlb_handle;

/* Fill *p with the defaults of BASELINE.json's literal physics (tau = tau_g = 1, rho0 = 1, G12 = 0.405,
 * G11a = G22a = -9, G11r = G22r = 8.1, rho_wall = 0.52, T_bottom = 1, T_top = 0, T_ref = 0.5,
 * alpha_g = 1e-4, walls in y, thermal on, no droplets). */
int tlb_default_params(tlb_params* p);

/* Bytes of device memory tlb_create needs for an nx x ny lattice (both population buffers with
 * their ghost rows, the solid mask, the boundary-link list, 5 field planes, reduction partials). */
int tlb_workspace_bytes(int nx, int ny, const tlb_params* p, size_t* bytes);

/* Create a handle on `workspace` (DEVICE pointer, >= tlb_workspace_bytes, 256-byte aligned, caller
 * owned) that enqueues all work on `stream` (a cudaStream_t passed as void*; NULL = default stream).
 * TLB_EINVAL: nx, ny < 1, tau or tau_g <= 1/2, rho0 <= 0, moving walls or posts with periodic_y (the paper's own
 * warning, footnote L302), 2*post_h >= ny, post_w > post_period, NULL pointers, workspace too small. */
int tlb_create(int nx, int ny, const tlb_params* p, void* workspace, size_t workspace_bytes,
               void* stream, tlb_handle** out);
int tlb_destroy(tlb_handle* h);

/* Y-slab handle for rows [y0, y1) of the nx x ny lattice (see Y-SLABS above).  TLB_EINVAL additionally for
 * y0 < 0, y1 > ny, y1 <= y0, or fewer than 3 owned rows next to a halo face. */
int tlb_slab_workspace_bytes(int nx, int ny, int y0, int y1, const tlb_params* p, size_t* bytes);
int tlb_create_slab(int nx, int ny, int y0, int y1, const tlb_params* p, void* workspace, size_t workspace_bytes,
                    void* stream, tlb_handle** out);
/* out6 = { ny_local, own0, own1, y_off, halo_lo, halo_hi }: owned local rows [own0, own1); local row r is row
 * y_off + r of the whole lattice (wrapped when periodic_y).  A whole-lattice handle reports {ny, 0, ny, 0, 0, 0}. */
int tlb_slab_layout(const tlb_handle* h, int32_t out6[6]);
/* Bytes of one packed halo face: 27 planes x 3 padded rows in the storage precision. */
int tlb_halo_bytes(const tlb_handle* h, size_t* bytes);
/* Rows per CTA segment of the fused kernel's launch (so that tests can aim at a segment edge). */
int tlb_seg_rows(const tlb_handle* h);

/* Seeded initial state of the input recipe: structured posts from params, n_droplets
 * discs by random sequential addition, +noise, linear T profile (L314), populations at rest
 * equilibrium f = w rho, g = w T (R14).  Bit-identical to inputs/__init__.py (the seeded generators next to oracle/). */
int tlb_init(tlb_handle* h, uint64_t seed);

/* The same with the paper's own droplet arrangement ("droplet initialisation = 1", L266: "we initialise the soft domains
 * in an honeycomb structure, where we establish the total number of droplets by calibrating the relative number of
 * droplets along x and y"): ndx x ndy discs of params.droplet_radius, row j at y = post_h + (j + 1/2)(ny - 2 post_h)/ndy,
 * column i at x = (i + 1/4 + (j mod 2)/2) nx/ndx.  Bit-identical to inputs.honeycomb_centres + inputs.initial_fields.
 * TLB_EINVAL for ndx, ndy < 1 or 2 ndx ndy > nx ny. */
int tlb_init_honeycomb(tlb_handle* h, int32_t ndx, int32_t ndy, uint64_t seed);

/* Rough walls with trapezoidal obstacles (section 4, Fig. 7(a), Table A.6; reading R27): replaces the obstacle
 * mask like tlb_set_solid (state and graphs are dropped).  An obstacle stands on the wall every `lambda` nodes; in row
 * j = 0 .. height - 1 counted from the wall it covers l(j) <= (x mod lambda) < width - r(j), r(j) = floor(j tan(alpha))
 * (alpha in radians, evaluated on the host), l(j) = r(j), or 0 when `asymmetric`; the top wall carries the y-mirror
 * image.  alpha = 0 gives the rectangular posts of tlb_params.  TLB_EINVAL with periodic_y, lambda < 1,
 * width > lambda, width or height < 0, obstacles of the two walls touching (2 height > ny). */
typedef struct tlb_rough_walls {
  double alpha;                         /* inclination of the trapezoid's side(s), radians; Table A.6: 0.25  */
  int32_t up, down;                     /* roughWallUp, roughWallDown                                          */
  int32_t width, height, lambda;        /* base width, height, period (nodes)                                  */
  int32_t asymmetric;                   /* 1: only the right-hand side is inclined                             */
} tlb_rough_walls;
int tlb_set_rough_walls(tlb_handle* h, const tlb_rough_walls* r);

/* Initial velocity perturbation (L322 "a finite perturbation is necessary to destabilise the conductive state",
 * Table A.5; reading R29): adds the roll pair du = (0, A sin(2 pi x/nx) sin(pi (y + 1/2)/ny)) to both fluids of the
 * current state, f_l,i += 3 w_i rho_l (c_i . du) on fluid sites (densities unchanged, momentum + rho_l du).  TLB_ESTATE
 * without a state. */
int tlb_perturb_velocity(tlb_handle* h, double amplitude);

/* Checkpoint files (Table C.11: "conf1_#.in / conf2_#.in / confG_#.in ... populations field dumped as a binary
 * file"; restart L324): <dir>/conf1_<index>.in, conf2_<index>.in, confG_<index>.in, each the raw little-endian fp64 array
 * [9][ny][nx] of tlb_get_populations (direction order R1; 0 on solid sites).  _read restores such a dump into a handle
 * of the same nx, ny (the obstacle mask is not part of a dump: set it first).  Synchronise; TLB_EIO on a file error. */
int tlb_write_checkpoint(tlb_handle* h, const char* dir, int32_t index);
int tlb_read_checkpoint(tlb_handle* h, const char* dir, int32_t index);

/* Field files of Tables C.9 / C.10 (L510-561) for the current state, written from the host after one read-back per field.
 * `what` is a sum of TLB_OUT_* flags; <i> = index:
 *   TLB_OUT_DENSITY      firstdensity.<i>.dat, seconddensity.<i>.dat      rho_A, rho_B
 *   TLB_OUT_TEMPERATURE  temperature.<i>.dat                              T
 *   TLB_OUT_VELOCITY     veloconf.<i>.dat, u_av.<i>.dat                   u^(H) (two columns), its x-average of u_x per row
 *   TLB_OUT_STRESS       Ptot_xy.<i>.dat, Pxy_av.<i>.dat                  P_xy (R21), its x-average per row
 *   TLB_OUT_ENERGY       timeEnergy.dat                                   one line "<i> E" APPENDED per call (L248: the kinetic
 *                                                                         energy E of tlb_observables "appended every nout
 *                                                                         energy steps"; pass the time step as index)
 * The paper names the files, not their format; reading R31: ASCII, one line "x y value" per site (velocity: "x y u_x
 * u_y"; the averages: "y value"), x fastest, a blank line after every lattice row, numbers printed with 17 significant
 * digits (they read back to the same doubles).  vtk != 0 adds <name>.<i>.vtk for the fields ("binary VTK 2.0", L244-246:
 * legacy "# vtk DataFile Version 2.0" header, BINARY, STRUCTURED_POINTS, one SCALARS / VECTORS array of big-endian doubles;
 * "write vtk file" of Table C.9).  Synchronises; TLB_EIO on a file error; TLB_EINVAL on slab handles. */
enum { TLB_OUT_DENSITY = 1, TLB_OUT_TEMPERATURE = 2, TLB_OUT_VELOCITY = 4, TLB_OUT_STRESS = 8, TLB_OUT_ENERGY = 16 };
int tlb_write_fields(tlb_handle* h, const char* dir, int32_t index, int32_t what, int32_t vtk);

/* Arbitrary obstacle mask [ny][nx], non-zero = solid (flag field, L286).  Resets the state. */
int tlb_set_solid(tlb_handle* h, const uint8_t* solid);
int tlb_set_solid_host(tlb_handle* h, const uint8_t* solid);

/* State from hydrodynamic fields: f_l,i = w_i rho_l, g_i = w_i T at rest (R14); solid sites ignored. */
int tlb_set_fields(tlb_handle* h, const double* rho_A, const double* rho_B, const double* T);
int tlb_set_fields_host(tlb_handle* h, const double* rho_A, const double* rho_B, const double* T);

/* State from / to time-t populations, each [9][ny][nx] (checkpoint / restart, L252).  tlb_get_populations(_host)
 * return TLB_ESTATE between tlb_slab_step_edges and tlb_slab_step_finish (the staging area is the buffer being written). */
int tlb_set_populations(tlb_handle* h, const double* fA, const double* fB, const double* g);
int tlb_get_populations(tlb_handle* h, double* fA, double* fB, double* g);
int tlb_set_populations_host(tlb_handle* h, const double* fA, const double* fB, const double* g);
int tlb_get_populations_host(tlb_handle* h, double* fA, double* fB, double* g);

/* Advance n >= 0 time steps (n = 0 is a no-op): per step one fused force+collide+stream kernel and
 * one wall/obstacle boundary kernel.  Whole blocks of 16 steps are replayed from a CUDA graph (one launch
 * instead of 32; matters for launch-bound lattices); the rest is launched kernel by kernel.  The graphs are
 * captured by the first call with n > 0 after the obstacle mask was set, before it enqueues anything.
 * TLB_EINVAL on a slab handle that has halo rows. */
int tlb_step(tlb_handle* h, int64_t n);

/* One time step of a y-slab in four parts (see Y-SLABS above); device pointers, all on the handle's stream.
 * face 0 = low y, 1 = high y; TLB_EINVAL for a face without halo rows.  While a step is open (after _edges,
 * before _finish) pack / unpack address the buffer being written, otherwise the current state.
 * TLB_ESTATE when called out of order. */
int tlb_slab_step_edges(tlb_handle* h);
int tlb_slab_step_interior(tlb_handle* h);
int tlb_slab_step_finish(tlb_handle* h);
int tlb_halo_pack(tlb_handle* h, int face, void* buf);
int tlb_halo_unpack(tlb_handle* h, int face, const void* buf);
/* Zero-copy alternative to pack / unpack: the population buffers keep the 27 plane rows of a lattice row next to one
 * another, so the 3 rows on either side of a face are ONE contiguous block of tlb_halo_bytes.  which = 0: the owned rows
 * next to `face` (what the neighbour imports); which = 1: the halo rows beyond `face` (where the neighbour's rows go).
 * *ptr is a DEVICE pointer into the buffer pack / unpack would address at this moment (the one being written while a
 * step is open); it changes from step to step (double buffer).  A transport (NCCL send / recv, a peer-to-peer copy, a
 * kernel of the neighbour storing through a peer mapping) can read the first and write the second directly, ordered
 * after tlb_slab_step_edges and before tlb_slab_step_finish on the handle's stream.  Same error codes as tlb_halo_pack. */
int tlb_halo_region(tlb_handle* h, int face, int which, void** ptr, size_t* bytes);

/* Measurement aid: advance ONE step, launching the fused kernel n (1..4096) times back to back on the
 * same input / output buffers and then the boundary kernel n times (both are idempotent on fixed inputs),
 * with CUDA events recorded on the handle's stream around each batch; returns the average duration in
 * milliseconds of one fused-kernel launch and of one boundary-kernel launch (HOST pointers).
 * Synchronises the stream. */
int tlb_profile_step(tlb_handle* h, int64_t n, double* fused_ms, double* boundary_ms);

/* Hydrodynamic fields at the current time: rho_A, rho_B [ny][nx], u = u^(H) [2][ny][nx] (L139),
 * T [ny][nx].  Any pointer may be NULL to skip that field. */
int tlb_fields(tlb_handle* h, double* rho_A, double* rho_B, double* u, double* T);
int tlb_fields_host(tlb_handle* h, double* rho_A, double* rho_B, double* u, double* T);

/* out[4] = { mass_A, mass_B, E, Nu }: mass_l = sum over fluid sites of rho_l (north_star);
 * E = mean over fluid sites of |u^(H)|^2 (L248, R11); Nu of Eq. (24) L347 in the reading R10.
 * tlb_observables writes to a DEVICE pointer; tlb_observables_host to a HOST pointer (synchronises).
 * One pass over the populations: the fused kernel reduces inside each CTA with warp shuffles, a second
 * small kernel combines the CTAs; fixed order, deterministic.  TLB_EINVAL on a slab handle with halo rows:
 * tlb_observable_sums writes the slab's share sums6 = { mass_A, mass_B, sum |u^(H)|^2, sum u_y^(H) T,
 * sum d_y T, fluid sites } (DEVICE), and tlb_observables_from_sums turns the all-reduced sums into out4. */
int tlb_observables(tlb_handle* h, double* out4);
int tlb_observables_host(tlb_handle* h, double* out4);
int tlb_observable_sums(tlb_handle* h, double* sums6);
int tlb_observables_from_sums(tlb_handle* h, const double* sums6, double* out4);

/* u_av[ny] (DEVICE pointer; _host: HOST pointer, synchronises): the x-average over the fluid sites of every
 * row of u_x^(H), the profile the paper dumps as u_av.dat for the Couette rheology (L248-250, Eq. (23));
 * 0 for a row without fluid sites.  Deterministic (one CTA per row, fixed-order sums). */
int tlb_x_average(tlb_handle* h, double* u_av);
int tlb_x_average_host(tlb_handle* h, double* u_av);

/* P_xy [ny][nx]: the off-diagonal component of the total stress (pressure-tensor sign: P_xy = -eta du_x/dy in a
 * simple shear) that the paper dumps as Ptot_xy.dat and, x-averaged over the fluid sites of each row, as
 * Pxy_av.dat [ny] for the rheology (L248-250, Eq. (23)).  The paper gives no formula; reading
 * R21: "the sum of all components contributions" (L296) =
 *   sum_l 1/2 sum_i c_ix c_iy (f_l,i + f*_l,i)                the momentum flux carried by the populations that
 *                                                             arrive at and leave the site (f*: post-collision)
 * + 1/2 sum_c c_x c_y [ G12 (psi^x_A(x) w(c) psi^x_B(x+c) + psi^x_B(x) w(c) psi^x_A(x+c))
 *                       + sum_l psi^s_l(x) (G_ll^a w(c) + G_ll^r p(c)) psi^s_l(x+c) ]   the interaction part of
 *                                                             Eqs. (7), (10), (11) (wall values at solid nodes).
 * 0 at solid sites.  Same conventions as tlb_fields / tlb_x_average. */
int tlb_stress_xy(tlb_handle* h, double* P_xy);
int tlb_stress_xy_host(tlb_handle* h, double* P_xy);
int tlb_x_average_stress(tlb_handle* h, double* Pxy_av);
int tlb_x_average_stress_host(tlb_handle* h, double* Pxy_av);

/* Droplet analysis, first stage (section 2.4; reading R22): bulk sites = fluid sites with rho_A > B_th;
 * droplets = clusters of nearest-neighbour (4-connected) bulk sites, x periodic (y too with periodic_y).
 *   labels     [ny][nx] int32 or NULL: smallest site index (y nx + x) of the site's cluster, -1 off the bulk
 *   n_droplets the number of droplets found
 *   stats      [max_droplets][4] = { label, sites, centre x, centre y } in ascending label order; the centre is
 *              the mean position of the cluster's sites (minimum image in x from the label site, wrapped to
 *              [0, nx)).  Meaningful only if n_droplets <= max_droplets.
 * Integer / index work: every output is bit-identical to the oracle's flood fill.  DEVICE pointers; _host: HOST
 * pointers (synchronises).  TLB_EINVAL on slab handles and for max_droplets > nx ny / 4. */
int tlb_droplets(tlb_handle* h, double B_th, int32_t* labels, int32_t max_droplets, int32_t* n_droplets, double* stats);
int tlb_droplets_host(tlb_handle* h, double B_th, int32_t* labels, int32_t max_droplets, int32_t* n_droplets, double* stats);

/* Droplet analysis, second stage (section 2.4, Eq. (25)).  The paper describes it in prose and defers
 * the details to its ref. [58]; readings R23-R26.  DEVICE pointers, asynchronous on the handle's stream,
 * integer outputs bit-identical to the oracle's brute force.  The calls use the handle's scratch planes (they do not
 * touch the populations); TLB_EINVAL on slab handles.
 *
 * tlb_voronoi (R23, "each point of the lattice is coloured by the label of the nearest centre of mass"):
 *   centres [n][2] = { x, y } (e.g. columns 2, 3 of tlb_droplets' stats), colour [ny][nx] int32 = index k of the centre
 *   with the smallest squared distance (x minimum image; y too with periodic_y), evaluated in fp64 without fused
 *   multiply-add; ties go to the smallest index; -1 everywhere for n = 0.  n <= nx ny / 4.
 * tlb_delaunay (R24, "The vertices at which adjacent digital Voronoi cells converge are used to identify the Delaunay
 *   triangulation"): a vertex is a 2 x 2 block of sites (x periodic; y periodic with periodic_y, else the rows beyond
 *   the flat walls carry a wall colour) holding >= 3 distinct colours; 3 colours link every pair of droplets in the
 *   block, 4 colours the four side pairs and the main-diagonal pair (x, y)-(x+1, y+1).  links [max_links][2], a < b,
 *   distinct, in lexicographic order; *n_links = their number (only the first max_links are written), or -1 if a
 *   droplet has more than 32 links.  n = number of colours (droplets).
 * tlb_droplet_match (R25): map[i] = colour_past at the site nearest to the present centre i (floor(c + 1/2), x wrapped,
 *   y wrapped or clamped): the past droplet in whose Voronoi cell the present droplet lies.
 * tlb_droplet_displacements (L326, L340: the "Lagrangian droplet displacement vector fields" of the deltaAnalysis output):
 *   disp[i] = X_i(now) - X_map[i](past) [n_now][2], minimum image in x (in y with periodic_y); (0, 0) where map[i] < 0.
 * tlb_t1_events (R25, "the diagonal link between a and b is replaced by the link between c and d"): both link lists as
 *   tlb_delaunay writes them; map (or NULL = identity; n_map entries) rewrites the ends of the present links into
 *   indices of the past frame (links with an end mapped to < 0 or both ends on one droplet are dropped); n_droplets =
 *   droplets of the past frame.  events [max_events][4] = { a, b, c, d }, a < b, c < d: a-b linked in the past and not
 *   now, c-d now and not in the past, the sides a-c, a-d, b-c, b-d in both; lexicographic order; *n_events = their
 *   number, or -1 on table overflow.
 * tlb_droplet_nusselt (R26, Eq. (25)): nu[i] = [u_y^(H) T - kappa d_y T] / (kappa dT / ny) at the site nearest to centre
 *   i, kappa and d_y T as in Eq. (24) / R10; 0 on a solid site.  TLB_ESTATE without a state. */
int tlb_voronoi(tlb_handle* h, const double* centres, int32_t n, int32_t* colour);
int tlb_delaunay(tlb_handle* h, const int32_t* colour, int32_t n, int32_t max_links, int32_t* n_links, int32_t* links);
int tlb_droplet_match(tlb_handle* h, const int32_t* colour_past, const double* centres_now, int32_t n_now, int32_t* map);
int tlb_droplet_displacements(tlb_handle* h, const double* centres_past, const double* centres_now, const int32_t* map,
                              int32_t n_now, double* disp);
int tlb_t1_events(tlb_handle* h, const int32_t* links_past, int32_t n_past, const int32_t* links_now, int32_t n_now,
                  const int32_t* map, int32_t n_map, int32_t n_droplets, int32_t max_events, int32_t* n_events,
                  int32_t* events);
int tlb_droplet_nusselt(tlb_handle* h, const double* centres, int32_t n, double* nu);

/* tlb_t1_events for callers that cannot allocate device memory.  Every other call of this library works inside the
 * workspace given to tlb_create, and tlb_t1_events keeps its adjacency tables there.  This variant needs no handle and
 * no workspace, and it makes no cudaMalloc / cudaFree or other allocating call, ever: its tables live in a fixed array
 * inside the library's device image (about 4.3 MB that every GPU which loads libtlb.so holds until the process ends).
 * It is meant for
 *   - tools that only compare two Delaunay link lists (the paper's deltaAnalysis, L338-341) and own no lattice;
 *   - a monitor called from inside a time loop whose lattice was sized to fill the GPU: an allocation there can fail,
 *     and even a successful cudaMalloc holds up all streams of the device while it runs;
 *   - code hosted by an application that manages all device memory itself and does not let guests allocate.
 * Arguments, outputs and their order are those of tlb_t1_events (R25, section 2.4) minus the handle: DEVICE
 * pointers owned by the caller, nothing retained; the work is enqueued on `stream` (a cudaStream_t as void*, NULL =
 * default stream) of the calling thread's CURRENT device and the call returns without synchronising.  The events are
 * bit-identical to tlb_t1_events'.
 * Limits: n_droplets <= TLB_T1_STATIC_MAX_DROPLETS, else TLB_ELIMIT and nothing is enqueued; if more than
 * TLB_T1_STATIC_MAX_EVENTS events are found, *n_events = -1 (as on a table overflow).  n_past, n_now, n_map and
 * max_events are not limited.
 * One array serves every call in the process on a given GPU.  Each call clears, on its stream, the part it relies on,
 * so consecutive calls on one stream are independent; two calls that may run at the same time on one GPU (different
 * streams, or different threads) overwrite each other's tables and give garbage: serialise them.
 * The first call on each device also loads the device code and looks the array up (cudaGetSymbolAddress); make that
 * call before any stream capture begins.
 * TLB_EINVAL for negative counts or missing pointers, TLB_ECUDA for a CUDA error (also one left pending by others). */
#define TLB_T1_STATIC_MAX_DROPLETS 16384
#define TLB_T1_STATIC_MAX_EVENTS 16384
int tlb_t1_events_static(const int32_t* links_past, int32_t n_past, const int32_t* links_now, int32_t n_now,
                         const int32_t* map, int32_t n_map, int32_t n_droplets, int32_t max_events, int32_t* n_events,
                         int32_t* events, void* stream);

/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
int64_t tlb_launch_count(const tlb_handle* h);

/* Message for a return code; cudaGetErrorString of the sticky CUDA error of a handle. */
const char* tlb_error_string(int code);
const char* tlb_last_cuda_error(const tlb_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* TLB_H */
