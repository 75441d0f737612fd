/* fargo_oracle.h -- C interface of the CPU ORACLE.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this library.  It is a plain, slow, single
 * threaded fp64 restatement of one full hydrodynamic update of the FARGO3D method, written from
 * /root/reference/PAPER.md ("P:n" = line n of that file) with the readings listed in DESIGN.md.
 * It shares no code with the CUDA path (paper_1602_02359_b200/csrc) and neither includes the other.
 *
 * PARITY PINS: tests/test_oracle_*.py (closed forms, invariants, the paper's worked figures, brute force; the list is
 * in DESIGN.md section 2).  PARITY UNPINNED -- conventions the paper leaves open and no closed form fixes, held only
 * by oracle <-> CUDA agreement: the boundary formulas (reading G22), the form of the potential (G12), C_0 of Eq. 73
 * (G10), C_q (G8; loosely pinned by the 2-3-zone Sod shock), when v0 is taken (G13), where the orbital step sits
 * (G14), PPA on q rather than Q (G17), the disk initial states.
 * Shearing sheet (geometry 3; Tab. 1/2 P:115; Eqs. 28-30; reading G32): pinned by the steady
 * shear flow, the epicyclic frequency and amplitude ratio, conservation of Tab. 2's X momentum and the exact
 * integer shift (tests/test_oracle_shearing_sheet.py).
 * MHD (NEXT-4; sections 3.6.1-3.7; mhd.cpp; readings G34-G37): pinned by v x B on uniform fields, div B and the mean
 * field to rounding, the Alfven phase speed along each axis, advection with the flow, pressure balance, the closed-form
 * pressure and tension accelerations, Eq. 115 (current sheet), the field-loop energy the paper prints at t = 2, and for
 * cell 11 the exact circular shift, the hydrodynamic orbital routine on B_Y and Eq. 94 (tests/test_oracle_mhd.py).
 * PARITY UNPINNED there: the ghost fill of B, the order inside cell 8 (G36), the extra ghost fill before it (G34).
 *
 * Layout of every field passed through this interface: nz*ny*nx doubles, X (i) fastest, ACTIVE
 * cells only; velocities on the LOWER face of the cell in their own direction.
 */
#ifndef FARGO_ORACLE_H
#define FARGO_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_CARTESIAN = 0, ORC_CYLINDRICAL = 1, ORC_SPHERICAL = 2,
       ORC_SHEARING_SHEET = 3 };  /* Tab. 1; shearing sheet: Cartesian metric */
enum { ORC_ISOTHERMAL = 0, ORC_ADIABATIC = 1 };                      /* Eqs. 6, 7 */
enum { ORC_PERIODIC = 0, ORC_OUTFLOW = 1, ORC_REFLECTING = 2 };

/* stages of one full update, in the order of Fig. 2 (caption P:198); see oracle_step_until */
enum {
  ORC_ST_BC1 = 0, ORC_ST_VMEAN, ORC_ST_POT, ORC_ST_DT, ORC_ST_SRC_A, ORC_ST_SRC_B, ORC_ST_SRC_C,
  ORC_ST_SRC_D, ORC_ST_BC2, ORC_ST_MOM, ORC_ST_SWEEP_X, ORC_ST_SWEEP_Y, ORC_ST_SWEEP_Z,
  ORC_ST_ORB_FRAC, ORC_ST_ORB_SHIFT, ORC_ST_NEWVEL, ORC_ST_COUNT
};

typedef struct oracle_mesh {
  int nx, ny, nz;            /* active cells; 1 = direction absent */
  double xmin, xmax;         /* uniform in X */
  const double* yedges;      /* ny+1 active edges, or NULL: uniform ymin + j*(ymax-ymin)/ny */
  const double* zedges;      /* nz+1 active edges, or NULL */
  double ymin, ymax, zmin, zmax;
  int bc[3][2];              /* [direction][lower, upper] */
  int nghost;                /* ghost layers, 3; 4 is accepted for the ghost-budget test */
} oracle_mesh;

typedef struct oracle_params {
  double gamma, cfl, cvnr2, nu;
  int fargo_on;
  double omega_frame, gm_star, planet_mass, planet_r, planet_phi0, planet_omega, planet_eps;
  double shear_c0, t_stop, dt_fixed;
  double oort_a;             /* Oort constant A of Eq. 29, shearing sheet only; Keplerian: -0.75 Omega_f */
} oracle_params;

typedef struct oracle_ctx oracle_ctx;

int oracle_init(oracle_ctx** out, const oracle_mesh* mesh, int geometry, int eos, const oracle_params* p);
int oracle_destroy(oracle_ctx* c);
int oracle_set_fields(oracle_ctx* c, const double* rho, const double* e, const double* vx,
                      const double* vy, const double* vz);
int oracle_get_fields(oracle_ctx* c, double* rho, double* e, double* vx, double* vy, double* vz);
/* NEXT-4, MHD on Cartesian meshes (sections 3.6.1-3.6.2; mhd.cpp; readings G34-G36): the face-centred
 * field (active cells; bx[i,j,k] on the LOWER X face of cell (i,j,k), like vx), mu0, the resistivity eta, and `passive`
 * (the field is transported and diffused but exerts no force: the current-sheet test).  Switches the MHD substeps on. */
int oracle_set_bfield(oracle_ctx* c, const double* bx, const double* by, const double* bz, double mu0, double eta, int passive);
int oracle_get_bfield(oracle_ctx* c, double* bx, double* by, double* bz);
double oracle_max_divb(oracle_ctx* c);
/* one MHD substep on the arrays as they stand: 0 ghost fill of B, 1 EMFs, 2 tension, 3 CT, 4 orbital advection of B */
int oracle_run_mhd_stage(oracle_ctx* c, int which);
int oracle_step(oracle_ctx* c, int n);
int oracle_get_time(oracle_ctx* c, double* t, double* last_dt, long long* nsteps);

/* NEXT-2, live planets (section 3.8; reading G33).  n <= ORC_MAX_PLANETS point masses: gm[p] = G m_p,
 * eps[p] = softening length of planet p's potential and of the gas force on it, pos/vel = 3n Cartesian components
 * in the frame rotating at omega_frame.  force_mode: 0 = the gas does not act on the planets, 1 = direct summation
 * over all cells, 2 = axisymmetric part of the density removed first; gconst = G.  With n > 0 the
 * fixed-orbit planet of oracle_params is ignored, the potential of cell 5 is that of the star and of these planets
 * where they are at the beginning of the update, and cell 5a (gas kick + one Cash-Karp step over dt, Eq. 109 with
 * Tab. 3) runs right after cell 6.  Cylindrical and spherical meshes only. */
#define ORC_MAX_PLANETS 8
int oracle_set_planets(oracle_ctx* c, int n, const double* gm, const double* eps, const double* pos,
                       const double* vel, int force_mode, double gconst);
/* returns n; gas_acc = the acceleration the gas gave each planet in the last update (3n) */
int oracle_get_planets(oracle_ctx* c, double* pos, double* vel, double* gas_acc);
/* test hooks: one Cash-Karp step of size h on the planets alone; sum_cells dm (x_c - x_p)/(d^2 + eps^2)^(3/2) for planet p */
/* Cell 5b, Eq. 44: the frame's rotation rate becomes omega_new between two updates; v_phi is corrected by
 * -(omega_new - omega_old) R_x(j,k) on every cell, live planets are carried into the new frame, the fixed-orbit
 * planet keeps its azimuth.  Cylindrical and spherical meshes (not the shearing sheet). */
int oracle_set_omega_frame(oracle_ctx* c, double omega_new);
/* Diagnostics (sum reductions): out[5] = mass, X / Y / Z momentum of Tab. 2 (mean of the left and right momenta
 * per cell; X = angular momentum on curvilinear meshes), internal energy (adiabatic).  Applies the ghost fill of cell 2. */
int oracle_diagnostics(oracle_ctx* c, double* out);
int oracle_planets_rk5(oracle_ctx* c, double h);
int oracle_gas_force(oracle_ctx* c, int p, double* F);

/* Run the NEXT update only up to and including `stage`, leaving intermediates in place.  The state
 * is then mid-step: inspect with oracle_get_array, do not call oracle_step afterwards. */
int oracle_step_until(oracle_ctx* c, int stage);
/* Run ONE stage on the arrays as they stand, with the current dt (oracle_set_dt overrides it). */
int oracle_run_stage(oracle_ctx* c, int stage);
int oracle_set_dt(oracle_ctx* c, double dt);
/* Copy a named internal array INCLUDING ghosts (TX*TY*TZ doubles, or TY*TZ for "v0"/"nshift").
 * names: rho e vx vy vz phi vxb vyb vzb vxc vyc vzc ec ed vxd vyd vzd pxm pxp pym pyp pzm pzp v0 nshift */
int oracle_get_array(oracle_ctx* c, const char* name, double* out);
int oracle_set_array(oracle_ctx* c, const char* name, const double* in);
int oracle_dims(oracle_ctx* c, int* tx, int* ty, int* tz, int* ngx, int* ngy, int* ngz);
/* Geometry tables (Tab. 5): surfaces of the lower faces and inverse volume of cell (j,k),
 * ghost-inclusive indices. */
int oracle_geometry(oracle_ctx* c, int j, int k, double* sx, double* sy, double* sz, double* invv,
                    double* lx, double* ly, double* lz);

/* 1-D primitives used by the sweeps, exposed so that tests can pin them to the paper's formulas. */
/* van Leer slopes a[m], m = 1..n-2, from cell values f and inverse centre distances
 * invd[m] = 1/(c_m - c_{m-1}); a[0] = a[n-1] = 0. */
void oracle_vanleer_slopes(int n, const double* f, const double* invd, double* a);
/* Upwind star value on the lower face of cell m, m = 1..n-1 (Eq. 48). */
void oracle_vanleer_star(int n, const double* f, const double* a, const double* len, const double* w,
                         double dt, double* fstar);
/* PPA star values on face i+1/2 of a periodic ring for a uniform shift of xi cells. */
void oracle_ppa_star(int n, const double* f, double xi, double* fstar);
/* PPA monotonised interface values fL, fR of a periodic ring (Eq. 71 + tests at P:484). */
void oracle_ppa_interfaces(int n, const double* f, double* fl, double* fr);

#ifdef __cplusplus
}
#endif
#endif
