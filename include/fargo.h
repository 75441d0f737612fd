/* fargo.h -- C ABI of the B200-native FARGO3D hydrodynamic timestep library (libfargo_b200.so).
 *
 * One full hydrodynamic update of the method of Benitez-Llambay & Masset, "FARGO3D: a new GPU-oriented
 * MHD code" (arXiv 1602.02359; "P:n" = line n of PAPER.md) on a structured staggered mesh, executed by
 * hand-written CUDA kernels for sm_100a.  One update is the sequence of Fig. 2 (caption P:198):
 *   ghost fill (cell 2) -> ring mean velocity (cell 3, Eq. 72) -> potential (cell 5)
 *   -> CFL time step (cell 6, Eq. 59; shear limit Eq. 73)
 *   -> source sub-steps 7a pressure/potential/centrifugal (Eqs. 27, 32-38, 53 P:245-280),
 *      7b von Neumann-Richtmyer viscosity, 7c compression work,
 *      7d viscous stress, 2-D cylindrical (App. B, Eqs. B2, B5 P:1160-1202)
 *   -> ghost fill (cell 9) -> momenta (12a, Eqs. 49-50)
 *   -> van Leer upwind sweeps X, Y, Z with consistent transport (12b-c, Eqs. 40-48)
 *   -> orbital advection: PPA fractional sweep + integer ring shift (Eqs. 60-71)
 *   -> new velocities (12d, Eq. 51).
 * The readings taken where the paper is silent or garbled are listed in DESIGN.md.
 *
 * There is NO CPU fallback: every call that needs the device fails with FARGO_ECUDA when no CUDA
 * device is usable.  Nothing throws across this boundary.  No global state: contexts are independent.
 *
 * FIELD LAYOUT for set/get: nz*ny*nx elements, X (index i) fastest, ACTIVE cells only, element type =
 * the context's precision (double for 64, float for 32).  vx[i,j,k] is v_X on the LOWER X face of cell
 * (i,j,k), vy on the lower Y face, vz on the lower Z face.  `e` is the internal energy
 * density (adiabatic, Eq. 7) or the sound-speed field c_s (isothermal, Eq. 6).
 * Directions are X,Y,Z = (x,y,z) | (phi,r,z) | (phi,r,theta) (Tab. 1).
 *
 * POINTERS: field pointers given to fargo_set_fields / fargo_get_fields may be HOST or DEVICE pointers
 * (resolved with cudaPointerGetAttributes).  mesh/params structs and table pointers inside them are
 * HOST memory, read during the call only.  `workspace` is DEVICE memory owned by the caller and must
 * stay alive, untouched, until fargo_destroy.  `cuda_stream` is a cudaStream_t (NULL = legacy default).
 */
#ifndef FARGO_B200_H
#define FARGO_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { FARGO_CARTESIAN = 0, FARGO_CYLINDRICAL = 1, FARGO_SPHERICAL = 2,
       FARGO_SHEARING_SHEET = 3 };   /* Tab. 1.  Shearing sheet (Tab. 2; Eqs. 28-30 P:249-255;
                                        DESIGN.md reading G32): the Cartesian mesh with X along the flow (periodic)
                                        and Y along the shear; needs nx > 1, ny > 1 and a periodic X axis */
enum { FARGO_ISOTHERMAL = 0, FARGO_ADIABATIC = 1 };                       /* Eqs. 6-7 */
enum { FARGO_PERIODIC = 0, FARGO_OUTFLOW = 1, FARGO_REFLECTING = 2,
       FARGO_EXTERNAL = 3 };   /* Y and Z faces: the ghosts beyond this face come from a neighbouring sub-domain (below) */

enum { FARGO_OK = 0, FARGO_EINVAL = -1, FARGO_ENOMEM = -2, FARGO_ECUDA = -3, FARGO_ESTATE = -4 };

/* Stages of one update, for fargo_step_until (per-kernel parity checks).  A fused kernel is observable
 * at the last stage it contains. */
enum {
  FARGO_ST_BC1 = 0, FARGO_ST_VMEAN, FARGO_ST_POT, FARGO_ST_DT, FARGO_ST_SRC_A, FARGO_ST_SRC_B,
  FARGO_ST_SRC_C, FARGO_ST_SRC_D, FARGO_ST_BC2, FARGO_ST_MOM, FARGO_ST_SWEEP_X, FARGO_ST_SWEEP_Y,
  FARGO_ST_SWEEP_Z, FARGO_ST_ORB_FRAC, FARGO_ST_ORB_SHIFT, FARGO_ST_NEWVEL, FARGO_ST_COUNT
};

typedef struct fargo_mesh {
  int nx, ny, nz;          /* active cells per direction; 1 = direction absent */
  double xmin, xmax;       /* X is uniform */
  const double* yedges;    /* HOST, ny+1 active cell edges, or NULL: uniform ymin + j*(ymax-ymin)/ny.  A slab (a Y face of
                              kind FARGO_EXTERNAL) must give them, preceded by the 3 edges beyond a cut lower face and
                              followed by the 3 edges beyond a cut upper face (the neighbouring slab's) */
  const double* zedges;    /* HOST, nz+1 active cell edges, or NULL (cut Z faces: as for yedges) */
  double ymin, ymax, zmin, zmax;
  int bc[3][2];            /* [direction][lower, upper]; X periodic => ghost-free wrapped X,
                              X non-periodic => 3 ghost layers in X too (reading G20) */
} fargo_mesh;

/* fargo_params.kernel_plan flags */
enum {
  FARGO_PLAN_UNFUSED_SOURCE = 1,   /* cells 7a-7c as k_source_a + k_source_b(c) instead of one pass */
  FARGO_PLAN_UNFUSED_VISC = 2,     /* cell 7d (3-D) as tensor + force kernels instead of one pass */
  FARGO_PLAN_UNFUSED_DT = 4,       /* cell 6 as its own pass instead of being folded into the previous update's last kernel */
  FARGO_PLAN_SEAM_ABOVE = 8        /* sub-domains: the upper FARGO_EXTERNAL Y face of this one is the periodic seam of the
                                      undivided mesh, whose first and last rings form no pair of Eq. 73 */
};

typedef struct fargo_params {
  double gamma;            /* adiabatic index (Eq. 7) */
  double cfl;              /* Courant number C of Eq. 59 (0.44) */
  double cvnr2;            /* C_q^2 of the artificial viscosity (reading G8; 2) */
  double nu;               /* constant kinematic viscosity, 0 = off (App. B) */
  int fargo_on;            /* orbital advection (section 3.5.1); needs periodic X */
  double omega_frame;      /* Omega_f (ignored in plain Cartesian geometry; constant in the sheet) */
  double gm_star;          /* G M of the central star (0 = none) */
  double planet_mass;      /* G m_p of the planet on a fixed circular orbit in the midplane (0 = none) */
  double planet_r, planet_phi0, planet_omega, planet_eps;   /* orbit radius, azimuth at t=0, angular
                              speed in the inertial frame, Plummer smoothing length (reading G12) */
  double shear_c0;         /* C_0 of Eq. 73 (0.5; reading G10) */
  double t_stop;           /* > 0: the step that would pass t_stop is clipped to land on it and later
                              steps are no-ops (reading G21); <= 0: none */
  double dt_fixed;         /* > 0: overrides the CFL time step */
  double oort_a;           /* Oort constant A of Eq. 29; shearing sheet only (Keplerian: -0.75 Omega_f) */
  int precision;           /* 64 (double) or 32 (float) */
  int use_graph;           /* 1: fargo_step replays one captured CUDA graph per update (needs a non-default
                              cuda_stream; on the legacy default stream it falls back to plain launches);
                              0: plain stream launches */
  int mhd;                 /* 1: reserve the arrays of the MHD substeps (NEXT-4: B, the EMFs, the star values, v_X - v0: 13 arrays);
                              they run once fargo_set_bfield has been called.  3-D meshes */
  int kernel_plan;         /* 0 = the fused kernels wherever they apply (default).  Bit flags select the unfused
                              sequences instead, for measurements and for tests that compare the two (results are
                              bit-identical): FARGO_PLAN_UNFUSED_SOURCE, FARGO_PLAN_UNFUSED_VISC, FARGO_PLAN_UNFUSED_DT */
  void* workspace;         /* DEVICE memory, >= fargo_workspace_bytes(), 256-byte aligned; caller-owned */
  size_t workspace_bytes;
  void* cuda_stream;       /* cudaStream_t on which every kernel and copy of this context is enqueued */
} fargo_params;

typedef struct fargo_ctx fargo_ctx;

/* Bytes of device workspace a context for (mesh, geometry, eos, params) needs.  0 on invalid input.
 * Does not touch the device. */
size_t fargo_workspace_bytes(const fargo_mesh* mesh, int geometry, int eos, const fargo_params* p);

/* Validate, build the Tab. 5 geometric coefficient tables and the trigonometric tables
 * on the host, upload them, carve the workspace.  On failure *out = NULL and a negative code is
 * returned; fargo_last_error(NULL) then describes the most recent init failure of this thread. */
int fargo_init(fargo_ctx** out, const fargo_mesh* mesh, int geometry, int eos, const fargo_params* p);
int fargo_destroy(fargo_ctx* c);

/* Load the five fields (layout above).  vy / vz may be NULL when that direction is absent.
 * Resets t = 0 and the step count.  Host pointers are copied through the context's stream. */
int fargo_set_fields(fargo_ctx* c, const void* rho, const void* e, const void* vx, const void* vy,
                     const void* vz);
/* Synchronise the stream and copy the active cells out (any pointer may be NULL = skip).  No
 * boundary fill is applied first. */
int fargo_get_fields(fargo_ctx* c, void* rho, void* e, void* vx, void* vy, void* vz);

/* Enqueue n full updates on the stream.  No host synchronisation inside.  (When the fixed-orbit planet moves in the
 * frame, planet_omega != omega_frame, every update carries one enqueued host node that forms the planet's position
 * from the device clock with the host's libm; the caller still does not wait and the update stays one graph.) */
int fargo_step(fargo_ctx* c, int n);

/* Synchronise and read the clock: simulated time, last time step, number of updates done. */
int fargo_get_time(fargo_ctx* c, double* t, double* last_dt, long long* nsteps);

/* Number of kernels launched (or replayed through graphs) by this context since fargo_init. */
long long fargo_kernel_launches(const fargo_ctx* c);

/* ---- inspection, for per-stage parity tests ---------------------------------------------------- */
/* Live planets (section 3.8; reading G33).  n <= FARGO_MAX_PLANETS point
 * masses around the star (gm_star of fargo_params, fixed at the origin).  All arrays are HOST, fp64, caller-owned:
 * gm[n] = G m_p; eps[n] = softening length of planet p's potential and of the gas force on it; pos[3n], vel[3n] =
 * Cartesian components in the frame rotating at omega_frame (constant).  force_mode: 0 = the gas does not act on the
 * planets, 1 = direct summation over all active cells, 2 = the axisymmetric part of the density is removed first
 * (P:717-720); gconst = G.  With n > 0 the fixed-orbit planet of fargo_params is ignored; every update then computes
 * the potential of cell 5 from the planets' current positions and, right after cell 6, runs cell 5a on the device:
 * v_p += dt a_gas(rho^n), then one fifth-order Cash-Karp step over dt (Eq. 109, Tab. 3).  The state
 * lives on the device: fargo_step(n) needs no host synchronisation.  Cylindrical and spherical meshes whose context
 * was created with a potential (gm_star != 0).  n = 0 switches back.  Errors: FARGO_EINVAL, FARGO_ESTATE, FARGO_ECUDA. */
#define FARGO_MAX_PLANETS 8
int fargo_set_planets(fargo_ctx* ctx, int n, const double* gm, const double* eps, const double* pos, const double* vel,
                      int force_mode, double gconst);
/* Synchronises the stream; copies positions, velocities and the acceleration the gas gave each planet in the last
 * update (3n each, HOST, any may be NULL).  Returns n (>= 0) or a negative error code. */
int fargo_get_planets(fargo_ctx* ctx, double* pos, double* vel, double* gas_acc);

/* Cell 5b, Eq. 44: from the next update on the frame rotates at omega_new.  v_phi is corrected by
 * -(omega_new - omega_frame) R_x(j,k) on every cell (R_x = r or r sin(theta) at the centre of the phi face), which
 * conserves angular momentum to rounding; live planets are carried into the new frame; the fixed-orbit planet keeps
 * its azimuth.  Host-initiated, between two fargo_step calls (it synchronises the stream; the paper does not say how
 * the new rate is chosen: DESIGN.md reading G33).  Cylindrical and spherical meshes only: FARGO_EINVAL otherwise. */
int fargo_set_omega_frame(fargo_ctx* ctx, double omega_new);

/* MHD (sections 3.6.1-3.6.2; readings G34-G36): method of characteristics +
 * constrained transport on 3-D meshes.  The context must have been created with fargo_params.mhd = 1.
 * bx, by, bz: the face-centred field, HOST or DEVICE, nz*ny*nx elements of the context's precision each, ACTIVE cells,
 * bx[i,j,k] on the LOWER X face of cell (i,j,k) like vx.  mu0 > 0; eta >= 0 is the resistivity of Eq. 5;
 * passive != 0: the field is transported and diffused but exerts no force (the current-sheet test).  From then on
 * every update also runs: the ghost fill of B (cell 2), C_w^2 = C_s^2 + v_A^2 and the resistive limit in Eq. 59 (cell 6),
 * the magnetic pressure gradient (cell 7a), star values and electromotive forces (cells 8a-8c, Eqs. 80-84), the
 * tension (cell 8d, Eq. 86), the constrained-transport update (cell 10, Eq. 76), which keeps div B to rounding, and, with
 * orbital advection on, the orbital advection of B by the upstream-averaged EMF (cell 11, section 3.7, Eqs. 92-107; the
 * substeps of cell 8 then see the residual velocity v_X - v0).
 * The source step then runs as the kernel sequence 7a, 7b(c) (the magnetic pressure enters before 7b).
 * On cylindrical and spherical meshes every length is the physical one at the place where it is used, Eq. 76 is applied with
 * the edge lengths and face areas of Tab. 5, and cell 7a gets the geometric terms of Eqs. 87-91 (reading G38).
 * fargo_get_bfield copies the active cells out (any pointer may be NULL).  Not on sub-domains; the resistive term on Cartesian
 * meshes only; the orbital advection of B not on spherical meshes: FARGO_EINVAL.  Errors: FARGO_EINVAL, FARGO_ESTATE, FARGO_ECUDA. */
int fargo_set_bfield(fargo_ctx* ctx, const void* bx, const void* by, const void* bz, double mu0, double eta, int passive);
int fargo_get_bfield(fargo_ctx* ctx, void* bx, void* by, void* bz);

/* Domain decomposition in Y and Z (section 4.1: the mesh is split in Y and Z, never
 * in X; 3 ghost layers are exchanged at cells 2 and 9 of Fig. 2; the time step is the minimum over the sub-domains,
 * P:407).  A sub-domain is an ordinary context whose mesh holds a range of rows / planes and whose cut faces have the
 * kind FARGO_EXTERNAL (with the neighbours' edges in yedges / zedges, see fargo_mesh).  fargo_step is refused on it;
 * one update is, on every sub-domain,
 *     exchange Y halos of the state -> fargo_update_phase(0)  cell 2: ghost fill of the faces that are not cut
 *     exchange Z halos of the state -> fargo_update_phase(1)  cells 3-6: v0, Phi, local dt
 *     all-reduce (min) of *fargo_dt_device_ptr -> fargo_update_phase(2)  t_stop flag retaken, source step (cell 7)
 *     exchange Y halos of (e, v)    -> fargo_update_phase(3)  cell 9
 *     exchange Z halos of (e, v)    -> fargo_update_phase(4)  transport, Eq. 51, clock
 * (Y before the fill and Z after it: the Z planes sent carry the Y ghosts, which is how the edges and corners travel.)
 * fargo_halo(which, dir, side, pack, buf): which = 0 the state (rho, e, vx, vy, vz), 1 = (e, vx, vy, vz) after the
 * source step; dir = 1 (Y, rows) or 2 (Z, planes); side = 0 lower / 1 upper face; pack != 0 copies the 3 ACTIVE layers
 * next to the face into buf, pack == 0 copies buf into the 3 GHOST layers beyond it.  buf is DEVICE memory of
 * fargo_halo_bytes(which, dir) bytes, caller-owned; what was packed on the lower side of a sub-domain is unpacked on the
 * upper side of the one below it, and vice versa (over NCCL, peer copies, or directly when both live on one device).
 * Everything is enqueued on the context's stream; no host synchronisation; with use_graph the kernels of each phase are
 * captured once and replayed.  The result is bit-identical to the
 * undivided mesh (tests/test_gpu_slabs.py).  Not with live planets.  Errors: FARGO_EINVAL, FARGO_ESTATE (phases out of
 * order), FARGO_ECUDA. */
int fargo_update_phase(fargo_ctx* ctx, int phase);
size_t fargo_halo_bytes(const fargo_ctx* ctx, int which, int dir);
int fargo_halo(fargo_ctx* ctx, int which, int dir, int side, int pack, void* device_buffer);
/* DEVICE address of the current time step (one double): all-reduce it in place (min) between phases 0 and 1. */
void* fargo_dt_device_ptr(fargo_ctx* ctx);
/* Sub-domains that live on ONE device: dt of this context <- min(dt, *other_dt_device_ptr), one tiny kernel on the context's
 * stream (the caller runs it pairwise over its sub-domains instead of an all-reduce; both contexts must share the stream). */
int fargo_dt_min_with(fargo_ctx* ctx, const void* other_dt_device_ptr);

/* Diagnostics, the sum reductions of P:787 ("the mass or angular momentum"): out[5] (HOST) = total mass, the X, Y and Z
 * momenta of Tab. 2 (per cell the mean of its left and right momenta, Eqs. 49-50; X is the angular
 * momentum on cylindrical and spherical meshes) and the internal energy (adiabatic; 0 otherwise), summed over the
 * active cells with the volumes of Tab. 5.  Applies the ghost fill of cell 2 first (the next update starts with the
 * same fill); synchronises the stream.  Reduced on the device in a fixed-shape tree: reproducible. */
int fargo_diagnostics(fargo_ctx* ctx, double* out);
/* The same sums for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): out_device[5] is a DEVICE address the caller owns; the call enqueues the ghost fill of cell 2, the
 * reduction kernel and a finishing kernel on the context's stream and returns WITHOUT synchronising (read out_device
 * after the stream has run).  It calls no cudaMalloc / cudaFree and no allocating routine: the per-block partial sums
 * live in a file-scope device array of the library (65536 x 5 doubles = 2.5 MiB, held by every device that loads the
 * library until exit), and are added on the device in block order, the order fargo_diagnostics adds them on the host.
 * Limit: ny * nz <= 524288 (8 rows along X per block); a larger mesh returns FARGO_EINVAL with a message and launches
 * nothing.  All contexts of a device share the array: calls that overlap on the GPU (different streams, no
 * dependency) race on it -- order them; the array's previous contents are never read.  The first call on a device
 * looks the array's address up (cudaGetSymbolAddress, which may load the module): make it once before a capture.
 * The device that holds the context's workspace must be current, as for every call. */
int fargo_diagnostics_noalloc(fargo_ctx* ctx, double* out_device);

/* Run the NEXT update up to and including `stage`; the state is then mid-step (only
 * fargo_get_array / fargo_dims / fargo_destroy / fargo_set_fields are valid afterwards). */
int fargo_step_until(fargo_ctx* c, int stage);
/* Ghost-inclusive extents and ghost counts of the device arrays. */
int fargo_dims(const fargo_ctx* c, int* tx, int* ty, int* tz, int* ngx, int* ngy, int* ngz);
/* Copy a named ghost-inclusive array (TZ*TY*TX elements of the context's precision, X fastest,
 * unpadded; TZ*TY for "v0") to HOST memory.  Names: rho e vx vy vz phi vxb vyb vzb vxc vyc vzc ec ed
 * vxd vyd pxm pxp pym pyp pzm pzp trho te v0 (MHD: bx by bz emfx emfy emfz).  pxm..pzp, trho, te refer to the transported set written
 * by the most recent transport pass.  Which names hold defined data depends on the stage reached. */
int fargo_get_array(fargo_ctx* c, const char* name, void* out);

/* ---- measurement ------------------------------------------------------------------------------------- */
/* enable != 0: from now on fargo_step uses plain launches and brackets every kernel launcher with a CUDA
 * event pair on the context's stream; enable == 0: stop and drop the record.  Either way the record restarts. */
int fargo_profile(fargo_ctx* c, int enable);
/* Synchronise, then write one text line per launcher into HOST buffer `buf` (len bytes):
 * "<name> <kernel launches> <total milliseconds>\n".  Names: bc vmean potential dt source_a source_b source_bc
 * source (7a-7c in one pass) source_d momenta sweep_x sweep_y sweep_z orbital newvel newvel_dt (Eq. 51 + the next update's per-cell CFL rate) advance. */
int fargo_profile_report(fargo_ctx* c, char* buf, size_t len);

/* Self-test of the branch-free fp64 division the kernels use in place of a / b (csrc/common.cuh, rdiv;
 * DESIGN.md "rounding"): out[n] = rdiv(a[n], b[n]) for n elements; a, b, out are DEVICE pointers to
 * doubles, `cuda_stream` a cudaStream_t (NULL = default stream).  b == NULL selects the kernels' division by
 * the constant six (rdiv6): out[n] = a[n] / 6.  Synchronises before returning.
 * Returns FARGO_OK or FARGO_ECUDA / FARGO_EINVAL (no context: message not retrievable). */
int fargo_selftest_div(const double* a, const double* b, double* out, long long n, void* cuda_stream);

/* Message for the last error of `c` (or of the last failed fargo_init on this thread when c == NULL). */
const char* fargo_last_error(const fargo_ctx* c);

#ifdef __cplusplus
}
#endif
#endif
